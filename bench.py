#!/usr/bin/env python
"""bench.py -- headline benchmark of the hot path (BASELINE.json: "energy+gradient evals/sec and ligands
docked/hour (1xB200) vs roofline").

One STEP = one pass of the whole hot path over one batch of synthetic
input: Lamarckian-GA docking of `--ligands` drug-like ligands (BASELINE.json configs[1]: 40 atoms, 8
rotatable bonds, 7 atom types, 9 fp32 maps of 64^3 at 0.375 A, 20 runs x population 150 x 2.5M evals per
run, ADADELTA on 6% of the individuals per generation) docked concurrently against one resident grid set
(row a7).  value = evaluations performed by all ranks / time.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--ligands L] [--impl reference]

Under torchrun every rank docks its own L ligands (the path shards by ligand with no exchange step:
"scaling": "weak"); time is the max over ranks.  `--impl reference` times the CPU oracle (test
infrastructure, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2007_03678_b200 import workloads as W  # noqa: E402

NRUN, POP, MAX_EVALS = 20, 150, 2_500_000
WORKLOAD = ("drug-like docking: 40-atom ligand, 8 torsions, 7 types, 9 fp32 maps 64^3 @0.375A, "
            "20 LGA runs x pop 150 x 2.5M evals/run, ADADELTA 300 it on 6%/generation")
FP32_LANES = 128                                            # per SM (B200_PROFILING.md unit counts)
L2_BYTES_PER_CLK = 6300.0                                   # LTS throughput cap of the full chip (B300_MICROARCH.md, measured on B300)
# one ligand = 20 runs x 9 ADADELTA chains = 180 chains = 6 groups of 32 lanes; the ADADELTA kernel keeps 12 warps (groups)
# resident per SM (positions in tensor memory) = 2 ligands; a step docks TWO waves of them, sorted by cost by the library, so
# that the hardware hands the next CTA to the SM that frees first (one wave: 5.80e8, two: 6.02e8 evals/s in that kernel)
LIGANDS_PER_SM = 4
# dram__bytes_read.sum + dram__bytes_write.sum of one dock_ls_lane_kernel launch on 148 SMs (profiles/r02b_dock_ls_lane_ncu.md:
# one `ncu --set full` capture each of `bench.py --probe dock <ligands> 0 40000`); other batches: null
LS_TRAFFIC_BYTES = {296: 2.6553e9 + 7.15e6, 592: 5.345e9 + 14.64e6}


def flops_per_eval(N, R, npairs, nmoved):
    """SURVEY.md section 8(d) op census (FMA = 2 FLOP): pose N*(30*dbar+30), grid N*150, pairs Np*100,
    back-prop N*20 + R*20; dbar = mean number of torsions acting on an atom."""
    dbar = nmoved / max(N, 1)
    return N * (30.0 * dbar + 30.0) + N * 150.0 + npairs * 100.0 + N * 20.0 + R * 20.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    return json.load(open(p)) if os.path.exists(p) else {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.idx = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.idx)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 8 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 8 and r[2].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            if len(r) >= 8:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def make_batch(L, rank):
    """grid set of configs[1] + L drug-like ligands (same shape, distinct seeds) for this rank"""
    grids, lig0 = W.make_config("drug")
    centre = 0.5 * (grids.box_lo + grids.box_hi)
    c = W.CONFIGS["drug"]
    ligs = [lig0 if (rank == 0 and i == 0) else W.make_ligand(c["N"], c["R"], c["T"], 1000 * rank + 100 + i, centre)
            for i in range(L)]
    return grids, W.share_type_table(ligs)                  # one force-field table for the batch, as in a screen


# ------------------------------------------------------------------------------------------ reference arm (CPU oracle)
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    grids, ligs = make_batch(1, 0)
    og, ol = oracle.Grids.from_workload(grids), oracle.Ligand.from_workload(ligs[0])
    par = oracle.params(W.DEFAULT_PARAMS)
    cores = oracle.num_threads()
    nrun = 2 * cores                                       # independent runs of the workload's ligand: every core stays busy
    sample_evals = 20_000                                  # per run; POP + k generations of (POP-1 + 9*300)
    sample = (f"oracle.dock (fp64, as it stands): 1 ligand of the workload x {nrun} runs x {sample_evals} evals/run on {cores} threads "
              f"(full budget: {NRUN} runs x {MAX_EVALS}); ratios against it are vs an unoptimised oracle")
    times, evals = [], 0
    for s in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = oracle.dock(og, ol, par, nrun, POP, sample_evals, seed=s)
        dt = time.perf_counter() - t0
        if s >= args.warmup:
            times.append(dt)
            evals += int(r["evals"].sum())
    total = sum(times)
    v = evals / total
    print(json.dumps({
        "impl": "reference", "metric": "energy+gradient evals/sec", "value": v, "unit": "evals/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / max(1, args.steps), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": v, "unit": "evals/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def reduce_over_ranks(dist, dev, times, counts):
    """Whole-job numbers from per-rank ones: times -> MAX over ranks, counts -> SUM over ranks (the path has no other
    collective: ranks dock disjoint ligand shards)."""
    import torch
    t = torch.tensor(list(times), dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(counts), dtype=torch.float64, device=dev)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist(), [int(x) for x in c.tolist()]


# ------------------------------------------------------------------------------------------ CUDA arm
def main():
    if "--probe" in sys.argv:
        return probe(sys.argv[sys.argv.index("--probe") + 1:])
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--ligands", type=int, default=0, help="ligands docked per step and per GPU (0: 4 per SM = two waves of the ADADELTA kernel)")
    ap.add_argument("--e2e-steps", type=int, default=1, help="steps of the host-buffer (end-to-end) leg, at most --steps")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip BASELINE.json configs[4] (adock_score_batch on the four sweep ligands)")
    ap.add_argument("--no-screen", action="store_true", help="skip configs[2] (virtual screen through adock_screen), configs[3] (large ligand) and the single-ligand call")
    ap.add_argument("--screen-ligands", type=int, default=10000)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2007_03678_b200 import binding as B

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    L = args.ligands if args.ligands > 0 else LIGANDS_PER_SM * sm_count
    grids, ligs = make_batch(L, rank)
    gp = B.make_params(W.DEFAULT_PARAMS)
    gg = B.Grids.from_workload(grids)
    gl = [B.Ligand.from_workload(gg, l, gp) for l in ligs]
    seeds = [10_000 * rank + i for i in range(L)]
    flop_eval = []
    for l, h in zip(ligs, gl):
        flop_eval.append(flops_per_eval(l.N, l.R, len(h.pairs()), int(h.tree()["moved"].sum())))
    l2_flush = torch.empty(160 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)     # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def step(s):
        return B.adock_dock_many(gg, gl, gp, NRUN, POP, MAX_EVALS, [sd + 1000 * s for sd in seeds])

    for s in range(args.warmup):
        l2_flush.zero_()
        step(s)
    # ---- device-resident timing: K steps, L2 flushed (outside the events) before each
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    B.adock_launch_count(reset=True)
    B.adock_profile(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    evals = 0
    for s in range(args.steps):
        l2_flush.zero_()
        ev[s][0].record()
        r = step(args.warmup + s)
        ev[s][1].record()
        evals += int(r["evals"].sum())
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = B.adock_launch_count()
    prof = B.adock_profile_read()
    dock_path = B.lib().adock_last_dock_path()
    B.adock_profile(False)
    t_ms = sum(a.elapsed_time(b) for a, b in ev)

    # ---- end to end through the C ABI with host buffers (adock_screen): per step = one batch of L ligands: host
    # preprocessing (R2) on worker threads + image upload from pinned memory (H2D), overlapped with the docking of the
    # previous batch, + docking + results (D2H); wall clock around the whole call
    barrier()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    host_threads = max(1, min(8, (os.cpu_count() or 2) - 1))
    e2e_ligs = ligs * e2e_steps
    e2e_seeds = [sd + 77 * (s + 1) for s in range(e2e_steps) for sd in seeds]
    t0 = time.perf_counter()
    r = B.adock_screen(gg, e2e_ligs, gp, NRUN, POP, MAX_EVALS, e2e_seeds, batch=L, host_threads=host_threads)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_evals = int(r["evals"].sum())
    screen_stats = r["stats"]
    h2d = sum(len(h.image()[0]) + len(h.lane_image()[0]) + 4 * h.N for h in gl) + 3 * 128 * L
    d2h = (r["genotypes"].nbytes + r["energies"].nbytes + r["evals"].nbytes) // e2e_steps

    if world > 1:
        (t_ms, e2e_s), (evals, e2e_evals, launches) = reduce_over_ranks(dist, dev, [t_ms, e2e_s], [evals, e2e_evals, launches])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = evals / (t_ms * 1e-3)
    peaks = measured_peaks()
    clk_mhz = float((clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0)
    alu = alu_peaks(B, sm_count, clk_mhz)
    # roofline of the dominant kernel (dock_ls_lane_kernel: ADADELTA chains, ~95 % of all evaluations, all energy + gradient)
    ls_ms, ls_n, ls_evals = prof["ls_ms"], prof["ls_launches"], prof["ls_evals"]
    mean_flop = float(np.mean(flop_eval))
    mean_atoms = float(np.mean([l.N for l in ligs]))
    ach_tf = (ls_evals * mean_flop / (ls_ms * 1e-3) / 1e12) if ls_ms > 0 else None
    kernel = "dock_ls_lane_kernel" if dock_path == 2 else "dock_ls_kernel"
    ls_rate = ls_evals / (ls_ms * 1e-3) if ls_ms > 0 else 0.0
    roofline = {"bound": "alu", "kernel": kernel, "achieved": ach_tf, "peak": alu["measured_tflops"], "unit": "TFLOP/s",
                "frac": (ach_tf / alu["measured_tflops"]) if ach_tf else None,
                "traffic": LS_TRAFFIC_BYTES.get(L) if (dock_path == 2 and sm_count == 148) else None,
                "peak_source": f"measured in this process by the library's FFMA2 microbenchmark (adock_alu_peak: {alu['measured_tflops']:.2f} TFLOP/s); "
                               f"derived {sm_count} SMs x {FP32_LANES} FP32 lanes x 2 x {clk_mhz:.0f} MHz = {alu['derived_tflops']:.2f} (B200_PROFILING.md); "
                               f"HBM ({peaks.get('hbm_gbs')} GB/s of measured) is not the bound: ~120 B per evaluation",
                "flop_per_eval": mean_flop, "avg_launch_ms": (ls_ms / ls_n) if ls_n else None, "launches_timed": ls_n,
                "evals_per_launch": (ls_evals / ls_n) if ls_n else None, "evals_per_s": ls_rate,
                # both candidate bounds of SURVEY.md section 8(d), evals/s; the smaller one is the denominator of `frac`
                "bounds_evals_per_s": roofline_bounds(alu["measured_tflops"], mean_flop, mean_atoms, sm_count, clk_mhz),
                "l2_gather_gbs": ls_rate * mean_atoms * 64.0 / 1e9}
    # every evaluation of the timed steps by kind: ADADELTA iterations are energy + gradient, the scoring of generation 0
    # and of the GA offspring is energy only
    eg = int(prof["ls_evals"])
    out = {
        "metric": "energy+gradient evals/sec", "value": value, "unit": "evals/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "ligands_per_step_per_gpu": L, "nrun": NRUN, "pop_size": POP, "max_evals": MAX_EVALS,
                   "l2": "160 MB buffer written before every timed step (flush); maps 113.8 MB re-laid-out",
                   "kernel_family": "lane-per-individual, positions in tensor memory" if dock_path == 2 else "warp-per-individual"},
        "evals": {"all": evals, "energy_gradient": eg * world if world == 1 else None, "energy_only": (evals - eg) if world == 1 else None,
                  "energy_gradient_per_s": eg / (t_ms * 1e-3) if world == 1 else None,
                  "note": "value counts every evaluation; energy_gradient = ADADELTA iterations (rank 0's count), energy_only = generation 0 + GA offspring"},
        "ligands_per_hour": 3600.0 * L * world * args.steps / (t_ms * 1e-3),
        "e2e": {"value": e2e_evals / e2e_s, "unit": "evals/s", "h2d_bytes_per_step": int(h2d) * world, "d2h_bytes_per_step": int(d2h) * world,
                "ligands_per_hour": 3600.0 * L * world * e2e_steps / e2e_s, "steps": e2e_steps,
                "api": "adock_screen (host buffers; preprocessing of batch b+1 overlapped with the docking of batch b)",
                "host_threads": host_threads, "host_prep_s": screen_stats["prep_s"], "host_exposed_s": screen_stats["exposed_s"],
                "gpu_idle_frac": max(0.0, 1.0 - screen_stats["dock_s"] / screen_stats["wall_s"])},
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
    }

    if not args.no_screen:
        out["virtual_screen"] = virtual_screen(B, torch, args.screen_ligands)
        out["large_ligand"] = large_ligand(B, torch, alu, sm_count, clk_mhz)
        # BASELINE.json configs[1] taken literally: ONE ligand per call (180 ADADELTA chains: a CTA of 4 warps per chain)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r1 = B.adock_dock(gg, gl[0], gp, NRUN, POP, MAX_EVALS, seed=4242, want_coords=True)
        dt1 = time.perf_counter() - t0
        out["single_ligand"] = {"workload": "configs[1] as one adock_dock call (1 ligand x 20 runs x 2.5M evals, host results)",
                                "seconds_per_ligand": dt1, "evals_per_s": float(r1["evals"].sum()) / dt1,
                                "ligands_per_hour": 3600.0 / dt1, "best_energy": float(r1["energies"].min())}
    if not args.no_sweep:
        out["score_batch"] = sweep(B, torch, dev, alu, sm_count, clk_mhz)
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline()
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def alu_peaks(B, sm_count, clk_mhz):
    """FP32 peak: measured by the library's FFMA2 microbenchmark in this process, and derived from unit counts and clock"""
    m = B.adock_alu_peak()
    return {"measured_tflops": float(m["tflops"]), "fma_lanes_per_clk_sm": float(m["fma_lanes_per_clk_sm"]),
            "derived_tflops": sm_count * FP32_LANES * 2 * clk_mhz * 1e6 / 1e12}


def roofline_bounds(peak_tflops, flop_eval, atoms, sm_count, clk_mhz):
    """the two candidate bounds in evaluations per second.  FP32: measured FFMA2 peak / algorithmic
    FLOP per evaluation.  L2 gather: the map lookups are 2 sector loads (2 x 32 B) per atom against the LTS throughput cap
    (B300_MICROARCH.md: ~6300 B/clk full chip, measured on B300; no B200 measurement in MEASURED_PEAKS.json)."""
    fp32 = peak_tflops * 1e12 / flop_eval
    l2 = L2_BYTES_PER_CLK * clk_mhz * 1e6 / (atoms * 64.0)
    return {"fp32": fp32, "l2_gather": l2, "binding": "fp32" if fp32 <= l2 else "l2_gather", "min": min(fp32, l2)}


def virtual_screen(B, torch, nlig):
    """BASELINE.json configs[2] (virtual-screen batch): `nlig` synthetic ligands (15-60 atoms, 0-15 torsions) against one
    shared 80^3 grid set, 10 runs x pop 150 x 250 k evals each, host buffers in and out through adock_screen (batches sized
    by the library; the next batch's preprocessing overlaps the current batch's docking).  Measured, not extrapolated."""
    grids, _ = W.make_config("screen")
    ligs = W.share_type_table(W.make_screen_ligands(nlig, grids, T=7, seed=2))
    gp = B.make_params(W.DEFAULT_PARAMS)
    gg = B.Grids.from_workload(grids)
    nrun, max_evals, batch = 10, 250_000, 0                 # batch 0: sized by the library
    threads = max(1, min(8, (os.cpu_count() or 2) - 1))
    nw = min(400, nlig)
    B.adock_screen(gg, ligs[:nw], gp, nrun, POP, 20_000, list(range(nw)), batch=0, host_threads=threads)     # warm-up
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    r = B.adock_screen(gg, ligs, gp, nrun, POP, max_evals, [7000 + i for i in range(nlig)], batch=batch, host_threads=threads)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    st = r["stats"]
    out = {"workload": f"{nlig} synthetic ligands (atoms 15-60, torsions 0-15), 9 maps 80^3 @0.375A, {nrun} runs x pop {POP} x "
                       f"{max_evals} evals, ADADELTA; adock_screen, {st['batches']} batches sized by the library, {threads} host threads",
           "ligands": nlig, "ligands_per_hour": 3600.0 * nlig / dt, "evals_per_s": float(r["evals"].sum()) / dt, "seconds": dt,
           "host_prep_s": st["prep_s"], "host_exposed_s": st["exposed_s"], "gpu_idle_frac": max(0.0, 1.0 - st["dock_s"] / st["wall_s"]),
           "best_energy_median": float(np.median(r["energies"].min(axis=1)))}
    gg.close()
    return out


def large_ligand(B, torch, alu, sm_count, clk_mhz):
    """BASELINE.json configs[3]: 128 atoms, 32 torsions, 8 types, 10 maps of 126^3, 50 runs x pop 150 x 2.5M evals, one
    adock_dock call with host results."""
    grids, lig = W.make_config("large")
    gp = B.make_params(W.DEFAULT_PARAMS)
    gg = B.Grids.from_workload(grids)
    gl = B.Ligand.from_workload(gg, lig, gp)
    fl = flops_per_eval(lig.N, lig.R, len(gl.pairs()), int(gl.tree()["moved"].sum()))
    B.adock_dock(gg, gl, gp, 50, POP, 60_000, seed=1)       # warm-up
    torch.cuda.synchronize()
    B.adock_profile(True)
    t0 = time.perf_counter()
    r = B.adock_dock(gg, gl, gp, 50, POP, MAX_EVALS, seed=3)
    dt = time.perf_counter() - t0
    pr = B.adock_profile_read()
    B.adock_profile(False)
    ev = float(r["evals"].sum())
    ls_rate = pr["ls_evals"] / (pr["ls_ms"] * 1e-3) if pr["ls_ms"] > 0 else None
    out = {"workload": "configs[3]: 128 atoms, 32 torsions, 8 types; 10 maps 126^3 @0.375A (1.0 GB re-laid-out, not L2-resident); 50 runs x pop 150 x 2.5M evals",
           "seconds_per_ligand": dt, "evals_per_s": ev / dt, "ligands_per_hour": 3600.0 / dt, "kernel_family": B.adock_last_dock_path(),
           "flop_per_eval": fl, "pairs": len(gl.pairs()), "ls_kernel_evals_per_s": ls_rate,
           "ls_kernel_alu_frac": (ls_rate * fl / 1e12 / alu["measured_tflops"]) if ls_rate else None,
           "l2_gather_gbs": (ls_rate * lig.N * 64.0 / 1e9) if ls_rate else None,
           "best_energy": float(r["energies"].min())}
    gl.close()
    gg.close()
    return out


def sweep(B, torch, dev, alu, sm_count, clk_mhz, configs=("sweep16", "sweep40", "sweep80", "sweep128")):
    """BASELINE.json configs[4]: adock_score_batch (energy + gradient) on 1k..1M random genotypes for the 16/40/80/128-atom
    ligands on a 64^3 grid set; per point evals/s, the FP32 fraction of the measured FFMA2 peak and the L2 gather rate
    (2 sectors of 32 B per atom and evaluation)."""
    gp = B.make_params(W.DEFAULT_PARAMS)
    out = {"alu_peak_tflops": alu["measured_tflops"], "l2_cap_gbs": L2_BYTES_PER_CLK * clk_mhz * 1e6 / 1e9}
    for cfg in configs:
        grids, lig = W.make_config(cfg)
        gg = B.Grids.from_workload(grids)
        gl = B.Ligand.from_workload(gg, lig, gp)
        fl = flops_per_eval(lig.N, lig.R, len(gl.pairs()), int(gl.tree()["moved"].sum()))
        res = {"atoms": lig.N, "torsions": lig.R, "pairs": len(gl.pairs()), "flop_per_eval": fl,
               "bounds_evals_per_s": roofline_bounds(alu["measured_tflops"], fl, lig.N, sm_count, clk_mhz)}
        for n in (1024, 16384, 262144, 1048576):
            G = torch.from_numpy(W.make_genotypes(n, lig.R, grids, seed=4)).to(dev)
            E = torch.zeros(n, device=dev)
            gr = torch.zeros((n, 6 + lig.R), device=dev)
            for _ in range(3):
                B.adock_score_batch(gg, gl, gp, G, E, None, gr)
            reps = 10 if n * lig.N <= 1048576 * 40 else 3
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                B.adock_score_batch(gg, gl, gp, G, E, None, gr)
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b) / reps
            rate = n / (ms * 1e-3)
            tf = rate * fl / 1e12
            res[str(n)] = {"ms": ms, "evals_per_s": rate, "tflops": tf, "alu_frac": tf / alu["measured_tflops"],
                           "l2_gather_gbs": rate * lig.N * 64.0 / 1e9, "l2_frac": rate * lig.N * 64.0 / (L2_BYTES_PER_CLK * clk_mhz * 1e6)}
        out[cfg] = res
        gl.close()
        gg.close()
    return out


def probe(argv):
    """Single-kernel-family timing runs (the commands the ncu captures under profiles/ are taken from):

        python bench.py --probe score <config> <n> <path> [reps]                       # adock_score_batch, energy + gradient
        python bench.py --probe dock <ligands> <path> [max_evals] [ls_method] [autostop]   # adock_dock_many, drug-like config
        python bench.py --probe large <path> [max_evals]                               # adock_dock, configs[3]
        python bench.py --probe screen <ligands> <batch>                               # adock_screen, configs[2] sample
        python bench.py --probe alu                                                    # adock_alu_peak
        python bench.py --probe tmem                                                   # adock_tmem_probe (tensor memory as per-lane scratch)

    <path> is the argument of adock_set_path: 0 auto, 1 warp per individual, 2 / 21 / 22 / 24 lane per individual
    (K chosen / 1 / 2 / 4 warps per group), 3 team per individual.  Prints one line; not the bench contract."""
    import torch
    from paper_2007_03678_b200 import binding as B
    mode = argv[0]
    dev = torch.device("cuda:0")
    if mode == "alu":
        print(B.adock_alu_peak(), flush=True)
    elif mode == "tmem":
        names = {1: "tensor memory, dependent tcgen05.ld.x1", 3: "shared memory, dependent LDS.32", 2: "tensor memory, 8 x tcgen05.ld.x2", 4: "shared memory, 8 x LDS.64"}
        for w in (4, 8, 12):
            r = B.adock_tmem_probe(w, 0)
            print(f"W={w:2d} write / read-back of every column (.x1, .x4 + .x2 at columns 6m): errors = {r['errors']}", flush=True)
            for m in (1, 3):
                print(f"W={w:2d} {names[m]:40s} {B.adock_tmem_probe(w, m)['cycles_per_iteration']:.1f} cycles per load", flush=True)
            for m in (2, 4):
                c = B.adock_tmem_probe(w, m)["cycles_per_iteration"]
                print(f"W={w:2d} {names[m]:40s} {c:.1f} cycles per 8 loads and warp = {w * 8 * 256 / c:.0f} B/clk/SM", flush=True)
    elif mode == "score":
        cfg, n, path = argv[1], int(argv[2]), int(argv[3])
        reps = int(argv[4]) if len(argv) > 4 else 10
        grids, lig = W.make_config(cfg)
        gp = B.make_params(W.DEFAULT_PARAMS)
        gg = B.Grids.from_workload(grids); gl = B.Ligand.from_workload(gg, lig, gp)
        B.lib().adock_set_path(path)
        G = torch.from_numpy(W.make_genotypes(n, lig.R, grids, seed=4)).to(dev)
        E = torch.zeros(n, device=dev); gr = torch.zeros((n, 6 + lig.R), device=dev)
        for _ in range(3):
            B.adock_score_batch(gg, gl, gp, G, E, None, gr)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            B.adock_score_batch(gg, gl, gp, G, E, None, gr)
        b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b) / reps
        print(f"score {cfg} n={n} path={path}: {ms:.4f} ms  {n/ms*1e3:.4g} evals/s", flush=True)
    elif mode == "screen":
        nlig, batch = int(argv[1]), int(argv[2])
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
              f"{p['ls_ms']:.0f} ms {p['ls_launches']} launches {p['ls_evals']/max(p['ls_ms'], 1e-9)*1e3:.3e} evals/s in-kernel; family "
              f"{B.lib().adock_last_dock_path()}", flush=True)
    elif mode in ("dock", "large"):
        if mode == "dock":
            L, path = int(argv[1]), int(argv[2])
            me = int(argv[3]) if len(argv) > 3 else MAX_EVALS
            lsm = int(argv[4]) if len(argv) > 4 else 0
            ast = int(argv[5]) if len(argv) > 5 else 0
            grids, lig0 = W.make_config("drug")
            centre = 0.5 * (grids.box_lo + grids.box_hi); c = W.CONFIGS["drug"]
            ligs = [W.make_ligand(c["N"], c["R"], c["T"], 100 + (0 if os.environ.get("ADOCK_PROBE_SAME_LIGAND") else i), centre) for i in range(L)]
            nrun = NRUN
        else:
            L, path = 1, int(argv[1])
            me = int(argv[2]) if len(argv) > 2 else MAX_EVALS
            lsm = ast = 0
            grids, lig0 = W.make_config("large")
            ligs, nrun = [lig0], 50
        gp = B.make_params(dict(W.DEFAULT_PARAMS, ls_method=lsm, autostop=ast))
        gg = B.Grids.from_workload(grids); gl = [B.Ligand.from_workload(gg, l, gp) for l in ligs]
        B.lib().adock_set_path(path)
        B.adock_dock_many(gg, gl, gp, nrun, POP, min(me, 100000), list(range(L)))
        B.adock_profile(True)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        r = B.adock_dock_many(gg, gl, gp, nrun, POP, me, [7 + i for i in range(L)])
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
        p = B.adock_profile_read()
        ev = int(r["evals"].sum())
        print(f"{mode} L={L} path={path} ls_method={lsm} autostop={ast} evals per run median {np.median(r['evals']):.0f} gens median "
              f"{np.median(r['gens']):.0f}: {dt:.3f} s {ev/dt:.4g} evals/s; ls kernel {p['ls_ms']:.1f} ms {p['ls_launches']} launches "
              f"{p['ls_evals']/max(p['ls_ms'], 1e-9)*1e3:.4g} evals/s in-kernel; family {B.adock_last_dock_path()}; "
              f"best E median {np.median(r['energies']):.3f}", flush=True)
    else:
        raise SystemExit(f"unknown probe mode {mode!r}")


def cpu_baseline():
    """The oracle as it stands (never tuned for this), timed on this box's host cores on bounded samples of the same
    workload: the whole LGA path (oracle.dock, fp64, runs spread over all cores: `value`), and the energy + gradient
    evaluation alone (oracle.score) in fp64 and in the honest-fp32 build, on one core and on all cores.  One warm-up and three
    repetitions each, best time.  A baseline, not the target: every ratio against it is `vs unoptimised oracle`."""
    import oracle
    grids, ligs = make_batch(1, 0)
    og, ol = oracle.Grids.from_workload(grids), oracle.Ligand.from_workload(ligs[0])
    par = oracle.params(W.DEFAULT_PARAMS)
    cores = oracle.num_threads()

    def best(fn, reps=3):
        fn()
        ts = []
        for _ in range(reps):
            t0 = time.perf_counter()
            fn()
            ts.append(time.perf_counter() - t0)
        return min(ts)

    nrun, sample_evals = 2 * cores, 20_000
    rr = {}
    def dock_all():
        rr["r"] = oracle.dock(og, ol, par, nrun, POP, sample_evals, seed=0)
    t_dock = best(dock_all)
    dock_evals = float(rr["r"]["evals"].sum())
    n1, nall = 2000, 2000 * cores
    G = W.make_genotypes(nall, ligs[0].R, grids, seed=11)
    legs = {}
    for name, fp32 in (("fp64", False), ("fp32", True)):
        t1 = best(lambda: oracle.score(og, ol, par, G[:n1], nthreads=1, fp32=fp32))
        ta = best(lambda: oracle.score(og, ol, par, G, nthreads=cores, fp32=fp32))
        legs[name] = {"evals_per_s_1_core": n1 / t1, "evals_per_s_all_cores": nall / ta}
    return {"value": dock_evals / t_dock, "unit": "evals/s", "cores": cores, "kind": "oracle",
            "sample": f"oracle.dock (fp64): 1 ligand of the workload x {nrun} runs x {sample_evals} evals/run on {cores} threads, best of 3 after "
                      f"a warm-up: {t_dock:.1f} s; oracle.score: {n1} (1 core) / {nall} (all cores) energy+gradient evaluations",
            "score_only": legs, "label": "vs unoptimised oracle"}


if __name__ == "__main__":
    main()
