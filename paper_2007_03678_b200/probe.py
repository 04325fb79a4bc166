"""Timing probe for one kernel family (used for the ncu captures under profiles/).

    python -m paper_2007_03678_b200.probe score <config> <n> <path> [reps]     # adock_score_batch, energy + gradient
    python -m paper_2007_03678_b200.probe dock <ligands> <path> [max_evals] [ls_method] [autostop]   # adock_dock_many, drug-like config

    python -m paper_2007_03678_b200.probe screen <ligands> <batch>                              # adock_screen, configs[2] sample

<path> is the argument of adock_set_path: 0 auto, 1 warp per individual, 2 / 21 / 22 / 24 lane per individual
(K chosen / 1 / 2 / 4 warps per group).  Needs a CUDA device."""
import sys
import time

import numpy as np
import torch

from . import binding as B, workloads as W


def main():
    mode = sys.argv[1]
    dev = torch.device("cuda:0")
    if mode == "score":
        cfg, n, path = sys.argv[2], int(sys.argv[3]), int(sys.argv[4])
        reps = int(sys.argv[5]) if len(sys.argv) > 5 else 10
        grids, lig = W.make_config(cfg)
        gp = B.make_params(W.DEFAULT_PARAMS)
        gg = B.Grids.from_workload(grids); gl = B.Ligand.from_workload(gg, lig, gp)
        B.lib().adock_set_path(path)
        G = torch.from_numpy(W.make_genotypes(n, lig.R, grids, seed=4)).to(dev)
        E = torch.zeros(n, device=dev); gr = torch.zeros((n, 6 + lig.R), device=dev)
        for _ in range(3): B.adock_score_batch(gg, gl, gp, G, E, None, gr)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps): B.adock_score_batch(gg, gl, gp, G, E, None, gr)
        b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b) / reps
        print(f"score {cfg} n={n} path={path}: {ms:.4f} ms  {n/ms*1e3:.4g} evals/s", flush=True)
    elif mode == "screen":
        nlig, batch = int(sys.argv[2]), int(sys.argv[3])
        grids, _ = W.make_config("screen")
        ligs = W.share_type_table(W.make_screen_ligands(nlig, grids, T=7, seed=2))
        gp = B.make_params(W.DEFAULT_PARAMS); gg = B.Grids.from_workload(grids)
        B.adock_screen(gg, ligs[:100], gp, 10, 150, 20000, list(range(len(ligs[:100]))), batch=0, host_threads=8)
        B.adock_profile(True)
        t0 = time.perf_counter()
        r = B.adock_screen(gg, ligs, gp, 10, 150, 250000, [7000 + i for i in range(nlig)], batch=batch, host_threads=8)
        dt = time.perf_counter() - t0
        p = B.adock_profile_read()
        print(f"screen n={nlig} batch={batch}: {dt:.2f} s {r['evals'].sum()/dt:.3e} evals/s batches {r['stats']['batches']} ls kernel "
              f"{p['ls_ms']:.0f} ms {p['ls_launches']} launches {p['ls_evals']/p['ls_ms']*1e3:.3e} evals/s in-kernel; family "
              f"{B.lib().adock_last_dock_path()}", flush=True)
    else:
        L, path = int(sys.argv[2]), int(sys.argv[3])
        me = int(sys.argv[4]) if len(sys.argv) > 4 else 2_500_000
        grids, lig0 = W.make_config("drug")
        centre = 0.5 * (grids.box_lo + grids.box_hi); c = W.CONFIGS["drug"]
        ligs = [W.make_ligand(c["N"], c["R"], c["T"], 100 + i, centre) for i in range(L)]
        lsm = int(sys.argv[5]) if len(sys.argv) > 5 else 0
        ast = int(sys.argv[6]) if len(sys.argv) > 6 else 0
        gp = B.make_params(dict(W.DEFAULT_PARAMS, ls_method=lsm, autostop=ast))
        gg = B.Grids.from_workload(grids); gl = [B.Ligand.from_workload(gg, l, gp) for l in ligs]
        B.lib().adock_set_path(path)
        B.adock_dock_many(gg, gl, gp, 20, 150, min(me, 100000), list(range(L)))
        B.adock_profile(True)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        r = B.adock_dock_many(gg, gl, gp, 20, 150, me, [7 + i for i in range(L)])
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
        p = B.adock_profile_read()
        ev = int(r["evals"].sum())
        print(f"dock L={L} path={path} ls_method={lsm} autostop={ast} evals per run median {np.median(r['evals']):.0f} gens median {np.median(r['gens']):.0f}: {dt:.3f} s {ev/dt:.4g} evals/s; ls kernel {p['ls_ms']:.1f} ms {p['ls_launches']} launches "
              f"{p['ls_evals']/p['ls_ms']*1e3:.4g} evals/s in-kernel; best E median {np.median(r['energies']):.3f}", flush=True)


if __name__ == "__main__":
    main()
