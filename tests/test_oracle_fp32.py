"""The oracle's compile-time fp32 mode ("to measure how far honest fp32 lands from fp64 -- sets
expectations for the GPU tolerance").  oracle/liboracle_f32.so is oracle/adock_oracle.cpp compiled with
-DORC_REAL=float: the score path (R3-R6) runs the SAME statements in float.  It is a measuring stick for the
tolerances of DESIGN.md R10, never the reference of a parity test.

What these tests establish (and print, so the numbers land in the test log):
  * on the NON-CLASHING workload honest fp32 sits well inside BASELINE.json's tolerances (energy
    1e-4 relative / 1e-3 absolute; gradient SURVEY C10 as written, no S_b term): median below 2 % of the tolerance,
    worst pose (an atom next to a clamped 1e5 map value) about a quarter of it;
  * on the clash-dominated random poses honest fp32 still meets the energy rule everywhere and the plain gradient rule
    on all but a fraction of a percent of the poses -- so the S_b term of R10 is a floor for rare poses, not a licence.
"""
import numpy as np
import pytest


def c10_plain(ref_grad, got_grad, R):
    """SURVEY C10 as written: per block ||d_b|| <= 1e-3 * max(||g_b||, 1e-2 ||g||) + 1e-4; returns err/tol [n, blocks]"""
    out = []
    gall = np.linalg.norm(ref_grad, axis=1)
    for lo, hi in ((0, 3), (3, 6), (6, 6 + R)):
        if hi == lo:
            continue
        d = np.linalg.norm(got_grad[:, lo:hi] - ref_grad[:, lo:hi], axis=1)
        tol = 1e-3 * np.maximum(np.linalg.norm(ref_grad[:, lo:hi], axis=1), 1e-2 * gall) + 1e-4
        out.append(d / tol)
    return np.stack(out, 1)


def test_fp32_build_is_a_separate_fp32_library(orc):
    assert orc.lib().orc_real_bytes() == 8 and orc.lib_f32().orc_real_bytes() == 4


@pytest.fixture(scope="module")
def pocket(W, orc):
    """non-clashing workload, CPU-sized: 20 atoms / 4 torsions, far_sep ligand, 40^3 maps with a pocket that fits it"""
    grids = W.make_grids(40, 4, 150, 7.0, seed=21)
    lig = W.make_ligand(20, 4, 4, seed=11, centre=0.5 * (grids.box_lo + grids.box_hi), far_sep=3.6, max_deg=3)
    return dict(grids=grids, lig=lig, og=orc.Grids.from_workload(grids), ol=orc.Ligand.from_workload(lig))


def test_nonclashing_workload_is_nonclashing(pocket, W, orc, par):
    c = pocket
    x = c["lig"].xyz.astype(np.float64)
    d = np.linalg.norm(x[c["ol"].pairs[:, 0]] - x[c["ol"].pairs[:, 1]], axis=1)
    assert d.min() >= 3.6 - 1e-6                        # no non-excluded pair starts inside its repulsive wall
    G = W.make_pocket_genotypes(1000, c["lig"].R, c["grids"], seed=5, sigma_t=0.7, sigma_tau=0.2)
    r = orc.score(c["og"], c["ol"], par, G)
    assert np.median(np.abs(r["E"])) < 1e3 and np.abs(r["terms"][:, 1]).max() < 50.0
    assert np.median(np.linalg.norm(r["grad"], axis=1)) > 1.0      # not a flat landscape either


def test_honest_fp32_on_nonclashing_poses(pocket, W, orc, par):
    c = pocket
    G = W.make_pocket_genotypes(1000, c["lig"].R, c["grids"], seed=5, sigma_t=0.7, sigma_tau=0.2)
    r64 = orc.score(c["og"], c["ol"], par, G)
    r32 = orc.score(c["og"], c["ol"], par, G, fp32=True)
    ok = (r64["margins"][:, 0] > 1e-3) & (r32["margins"][:, 0] > 1e-3)
    eratio = np.abs(r32["E"] - r64["E"]) / np.maximum(1e-4 * np.abs(r64["E"]), 1e-3)
    gratio = c10_plain(r64["grad"], r32["grad"], c["lig"].R)[ok]
    print(f"honest fp32, non-clashing: energy err/tol max {eratio.max():.4f}; gradient err/tol max {gratio.max():.4f}")
    assert eratio.max() < 0.5 and gratio.max() < 0.5 and np.median(eratio) < 0.02 and np.median(gratio) < 0.02


def test_honest_fp32_on_clash_poses(mid, W, orc, par):
    """the random poses of the BASELINE.json configs (median |E| ~ 3e6 kcal/mol)"""
    c = mid
    R = c["lig"].R
    G = W.make_genotypes(1000, R, c["grids"], seed=3)
    r64 = orc.score(c["og"], c["ol"], par, G)
    r32 = orc.score(c["og"], c["ol"], par, G, fp32=True)
    ok = (r64["margins"][:, 0] > 1e-3) & (r64["margins"][:, 1] > 1e-3) & (r32["margins"][:, 0] > 1e-3)
    eratio = np.abs(r32["E"] - r64["E"]) / np.maximum(1e-4 * np.abs(r64["E"]), 1e-3)
    gratio = c10_plain(r64["grad"], r32["grad"], R)[ok]
    frac_over = (gratio > 1.0).any(axis=1).mean()
    # the R10 rule with the S_b floor, for comparison
    sb = []
    for b, (lo, hi) in enumerate(((0, 3), (3, 6), (6, 6 + R))):
        d = np.linalg.norm(r32["grad"][:, lo:hi] - r64["grad"][:, lo:hi], axis=1)
        sb.append(d / (1e-3 * np.linalg.norm(r64["grad"][:, lo:hi], axis=1) + 1e-5 * r64["scales"][:, b] + 1e-4))
    sb = np.stack(sb, 1)[ok]
    print(f"honest fp32, clash poses: energy err/tol max {eratio.max():.3f}; plain C10 gradient rule exceeded on "
          f"{100 * frac_over:.2f} % of poses (worst {gratio.max():.2f}x); with the S_b floor worst {sb.max():.3f}x")
    assert eratio.max() < 1.0
    assert frac_over < 0.01 and gratio.max() < 5.0
    assert sb.max() < 0.25
