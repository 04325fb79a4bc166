"""N > 1 path on CPU: two gloo ranks dock disjoint ligand shards (no data-path collective) and the
whole-job numbers are reduced the way bench.py does it.  The docking itself is done by the CPU oracle here (test
infrastructure); the GPU library is exercised by tests/test_gpu_parity.py."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NLIG, NRUN, POP, EVALS = 5, 2, 8, 200


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _dock_ligands(indices):
    import oracle
    from paper_2007_03678_b200 import workloads as W
    grids, _ = W.make_config("tiny")
    c = W.CONFIGS["tiny"]
    centre = 0.5 * (grids.box_lo + grids.box_hi)
    og = oracle.Grids.from_workload(grids)
    par = oracle.params(dict(W.DEFAULT_PARAMS, lsit=10))
    out = {}
    for i in indices:
        lig = W.make_ligand(c["N"], c["R"], c["T"], 500 + i, centre)
        r = oracle.dock(og, oracle.Ligand.from_workload(lig), par, NRUN, POP, EVALS, seed=i)
        out[i] = (r["energies"].tolist(), int(r["evals"].sum()))
    return out


def _rank_main(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    from paper_2007_03678_b200 import workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = W.shard(NLIG, rank, world)
    res = _dock_ligands(mine)
    evals = sum(v[1] for v in res.values())
    t_ms = 10.0 * (rank + 1)                               # stand-in device time: rank 1 is the slow one
    (t_max, e_max), (evals_all, nlig_all) = bench.reduce_over_ranks(dist, torch.device("cpu"), [t_ms, 0.5 * t_ms], [evals, len(mine)])
    gathered = [None] * world
    dist.all_gather_object(gathered, res)
    dist.barrier()
    if rank == 0:
        q.put(dict(t_max=t_max, e_max=e_max, evals_all=evals_all, nlig_all=nlig_all, gathered=gathered))
    dist.destroy_process_group()


def test_two_gloo_ranks_dock_disjoint_shards_and_reduce(orc):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    serial = _dock_ligands(range(NLIG))
    merged = {}
    for part in got["gathered"]:
        assert not (set(part) & set(merged)), "shards overlap"
        merged.update(part)
    assert sorted(merged) == list(range(NLIG))
    for i in range(NLIG):                                  # a ligand's result does not depend on which rank docked it
        assert merged[i][1] == serial[i][1]
        assert np.array_equal(np.asarray(merged[i][0]), np.asarray(serial[i][0]))
    assert got["t_max"] == 20.0 and got["e_max"] == 10.0   # MAX over ranks
    assert got["evals_all"] == sum(v[1] for v in serial.values()) and got["nlig_all"] == NLIG   # SUM over ranks


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


@pytest.mark.parametrize("steps", [1])
def test_reference_arm_prints_the_contract_line(steps):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", str(steps), "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "evals/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["steps"] == steps and line["higher_is_better"] is True
