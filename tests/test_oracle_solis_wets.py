"""Pins for the oracle's Solis-Wets local search (R11; PAPER.md lines 58, 64, 136 name the method and cite
Solis & Wets 1981 [27]) and for autostop (R12).  The paper prints no worked example of either, so
the pins are closed forms of the published rule: every-trial-fails and every-trial-succeeds schedules of the step
scale, the first two steps written out from the Philox words, convergence on convex quadratics, and the invariants of
the docking variant.
"""
import math

import numpy as np
import pytest


def _par(orc, W, **kw):
    d = dict(W.DEFAULT_PARAMS, ls_method=1)
    d.update(kw)
    return orc.params(d)


def _xi(orc, seed, id, gen, it, D):
    """the 2u-1 variates of iteration `it`: word d&3 of draw (it*ceil(D/4) + d/4, purpose 6, id, gen)"""
    nq = (D + 3) // 4
    key = np.array([seed & 0xFFFFFFFF, seed >> 32], np.uint32)
    ctr = np.array([[it * nq + q, 6, id, gen] for q in range(nq)], np.uint32)
    w = orc.philox(key, ctr).reshape(-1)[:D]
    return 2.0 * ((w >> 8).astype(np.float64) / 16777216.0) - 1.0


def test_constant_function_contracts_to_the_lower_bound(orc, W):
    """no trial is ever strictly better: two evaluations per iteration, rho halves every 4 iterations, and the search
    ends when rho = 2^-7 < 0.01: 28 iterations, 56 evaluations, x untouched."""
    par = _par(orc, W, lsit=300)
    x0 = np.array([1.0, -2.0, 3.0])
    x, E, ev, it, rho, tr = orc.solis_wets_rn(x0, 5.0, lambda x: 5.0, np.ones(3), par, seed=3, id=1, gen=2)
    assert (it, ev) == (28, 56)
    assert rho == 2.0 ** -7
    assert np.array_equal(x, x0) and E == 5.0
    assert np.all(tr[:28] == 5.0) and np.isnan(tr[28:]).all()


def test_linear_function_always_succeeds_and_expands(orc, W):
    """on f = a.x one of x+delta, x-delta is strictly better (a.delta != 0): every iteration succeeds, rho doubles
    every 4 iterations, E decreases strictly, and evals = iterations + number of failed first trials."""
    a = np.array([1.0, -2.0, 0.5, 3.0, -1.5])
    par = _par(orc, W, lsit=12)
    f = lambda x: float(a @ x)
    calls = []
    x, E, ev, it, rho, tr = orc.solis_wets_rn(np.zeros(5), 0.0, lambda x: (calls.append(x), f(x))[1], np.ones(5), par, 7, 0, 1)
    assert it == 12 and rho == 8.0
    assert np.all(np.diff(np.concatenate([[0.0], tr[:12]])) < 0)
    assert ev == len(calls) and 12 <= ev <= 24
    assert math.isclose(E, f(x), rel_tol=1e-14)


def test_first_two_steps_closed_form(orc, W):
    """iteration 0: delta = rho0*amp*xi (bias 0), accepted with the sign that lowers f = a.x;
    iteration 1: delta = rho0*amp*xi' + gain*(+-delta0)... the bias follows the accepted direction."""
    a = np.array([2.0, -1.0, 0.25, 4.0, 1.0, -3.0])
    amp = np.array([2.0, 2.0, 2.0, 0.5, 0.5, 0.5])
    seed, id, gen = 0x1234567890, 17, 3
    f = lambda x: float(a @ x)
    x1, *_ = orc.solis_wets_rn(np.zeros(6), 0.0, f, amp, _par(orc, W, lsit=1), seed, id, gen)
    d0 = amp * _xi(orc, seed, id, gen, 0, 6)
    s0 = 1.0 if a @ d0 < 0 else -1.0
    assert np.allclose(x1, s0 * d0, rtol=0, atol=1e-15)
    x2, *_ = orc.solis_wets_rn(np.zeros(6), 0.0, f, amp, _par(orc, W, lsit=2), seed, id, gen)
    b = float(np.float32(0.4)) * s0 * d0                     # keep*0 + gain*(accepted step); params are float32 values
    d1 = amp * _xi(orc, seed, id, gen, 1, 6) + b
    s1 = 1.0 if a @ d1 < 0 else -1.0
    assert np.allclose(x2, s0 * d0 + s1 * d1, rtol=0, atol=1e-14)


def test_failure_halves_the_bias(orc, W):
    """f = |x|^2 from the minimiser: iteration 0 fails both ways (bias stays 0); from a point where the first step
    succeeded, a following double failure multiplies the bias by decay -- seen through the next proposal."""
    par = _par(orc, W, lsit=1)
    x, E, ev, it, rho, _ = orc.solis_wets_rn(np.zeros(4), 0.0, lambda x: float(x @ x), np.ones(4), par, 5, 2, 9)
    assert ev == 2 and it == 1 and np.array_equal(x, np.zeros(4)) and E == 0.0


@pytest.mark.parametrize("cond", [1.0, 30.0])
def test_converges_on_convex_quadratic(orc, W, cond):
    rng = np.random.default_rng(4)
    n = 6
    lam = np.geomspace(1.0, cond, n)
    Q = np.linalg.qr(rng.normal(size=(n, n)))[0]
    A = Q @ np.diag(lam) @ Q.T
    xs = rng.normal(size=n)
    f = lambda x: float(0.5 * (x - xs) @ A @ (x - xs))
    x0 = xs + rng.normal(size=n) * 3
    par = _par(orc, W, lsit=600, sw_rho_lb=1e-6)
    x, E, ev, it, rho, tr = orc.solis_wets_rn(x0, f(x0), f, np.ones(n), par, 11, 0, 0)
    assert E <= 1e-3 * f(x0)
    assert np.all(np.diff(tr[:it]) <= 0)                      # accepted energies never increase
    assert it <= ev <= 2 * it


def test_docking_variant_invariants(mid, orc, W):
    """never worse than the carried energy, evals in [it, 2 it], unit quaternion, wrapped torsions, reported energy =
    score of the reported genotype, and a different (id, gen) gives a different trajectory."""
    grids, lig, og, ol = mid["grids"], mid["lig"], mid["og"], mid["ol"]
    par = _par(orc, W, lsit=100)
    G = W.make_genotypes(6, lig.R, grids, seed=21).astype(np.float64)
    E0 = orc.score(og, ol, par, G, want_grad=False)["E"]
    outs = []
    for i in range(6):
        g, E, ev, it, rho, tr = orc.solis_wets(og, ol, par, G[i], E0[i], seed=9, id=i, gen=1)
        assert E <= E0[i] and it <= ev <= 2 * it and it <= 100
        assert abs(np.linalg.norm(g[3:7]) - 1) < 1e-12 or np.array_equal(g, G[i])
        assert (g[7:] >= -math.pi).all() and (g[7:] < math.pi + 1e-12).all()
        chk = orc.score_f64(og, ol, par, g, want_grad=False)[0]
        assert math.isclose(chk, E, rel_tol=1e-12, abs_tol=1e-12)
        outs.append(E)
    assert sum(e < e0 for e, e0 in zip(outs, E0)) >= 5       # clashing random poses: the search finds better ones
    g2, E2, *_ = orc.solis_wets(og, ol, par, G[0], E0[0], seed=9, id=77, gen=1)
    assert E2 != outs[0]


def test_dock_with_solis_wets_accounting_and_bowl(W, orc):
    """full LGA with Solis-Wets on the bowl maps (E = N k |centroid - centre|^2 + const for a rigid ligand): every
    run finds the minimiser; evals accounting: P + gens (P-1) <= evals <= P + gens (P-1 + n_ls 2 lsit)."""
    n, T, h = 40, 2, 0.375
    centre = 0.5 * (n - 1) * h
    ax = np.arange(n) * h - centre
    bowl = 0.05 * (ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2)
    maps = np.zeros((T + 2, n, n, n), np.float32); maps[:T] = bowl
    lig = W.make_ligand(10, 0, T, seed=5, centre=(centre,) * 3)
    og = orc.Grids(maps, h, np.zeros(3, np.float32)); ol = orc.Ligand.from_workload(lig)
    par = _par(orc, W, lsit=60)
    r = orc.dock(og, ol, par, nrun=4, pop_size=30, max_evals=8000, seed=2)
    assert np.abs(r["genotypes"][:, :3] - centre).max() < 0.15
    gens, ev = r["gens"], r["evals"]
    assert ((ev >= 30 + gens * 29) & (ev <= 30 + gens * (29 + 2 * 2 * 60))).all()


# ------------------------------------------------------------------------------- R12 autostop
def _bowl(W, orc):
    n, T, h = 40, 2, 0.375
    centre = 0.5 * (n - 1) * h
    ax = np.arange(n) * h - centre
    bowl = 0.05 * (ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2)
    maps = np.zeros((T + 2, n, n, n), np.float32); maps[:T] = bowl
    lig = W.make_ligand(10, 0, T, seed=5, centre=(centre,) * 3)
    return orc.Grids(maps, h, np.zeros(3, np.float32)), orc.Ligand.from_workload(lig), centre


def test_autostop_limits(W, orc):
    """as_tol = +large: the std-dev test passes as soon as the window is full, so every run ends at generation
    as_window exactly; as_tol = 0: std < 0 never holds, so the result equals the run without autostop."""
    og, ol, _ = _bowl(W, orc)
    base = dict(W.DEFAULT_PARAMS, lsit=20)
    r_inf = orc.dock(og, ol, orc.params(dict(base, autostop=1, as_window=5, as_tol=1e30)), 3, 20, 10 ** 6, seed=4)
    assert (r_inf["gens"] == 5).all()
    r_off = orc.dock(og, ol, orc.params(dict(base, max_gens=12)), 3, 20, 10 ** 6, seed=4)
    r_zero = orc.dock(og, ol, orc.params(dict(base, max_gens=12, autostop=1, as_window=5, as_tol=0.0)), 3, 20, 10 ** 6, seed=4)
    assert np.array_equal(r_off["energies"], r_zero["energies"]) and np.array_equal(r_off["gens"], r_zero["gens"])
    assert (r_off["gens"] == 12).all()


def test_autostop_ends_converged_runs_early(W, orc):
    """on the bowl every run converges within a few generations; with autostop it ends long before the eval budget,
    at the same minimiser, and the best-energy history's last as_window entries have std < as_tol."""
    og, ol, centre = _bowl(W, orc)
    d = dict(W.DEFAULT_PARAMS, lsit=60, autostop=1, as_window=6, as_tol=0.01)
    r = orc.dock(og, ol, orc.params(d), nrun=4, pop_size=30, max_evals=200000, seed=2, hist_len=400)
    assert (r["evals"] < 200000).all() and (r["gens"] >= 6).all()
    assert np.abs(r["genotypes"][:, :3] - centre).max() < 0.1
    for k in range(4):
        h = r["history"][k][1:r["gens"][k] + 1]              # entry 0 is the initial population
        assert np.std(h[-6:]) < 0.01
        if r["gens"][k] > 6:
            assert np.std(h[-7:-1]) >= 0.01                  # it did not qualify one generation earlier
