"""Pins for the oracle's scoring function: grid term (R4), intramolecular pair term (R5),
totals and gradient back-propagation (R6).  PAPER.md line 58 names the energy terms and line 116 the
three map kinds; nothing numeric is printed in the paper, so every pin is a closed form, an
invariant, a library special case, brute force, or a finite difference.
"""
import math

import numpy as np
import pytest
from scipy.ndimage import map_coordinates
from scipy.sparse import csr_matrix
from scipy.sparse.csgraph import shortest_path


# ------------------------------------------------------------------------------- R4 grid term
def test_trilinear_exact_at_nodes(tiny):
    g, og = tiny["grids"], tiny["og"]
    rng = np.random.default_rng(0)
    idx = rng.integers(0, 24, (200, 3))
    idx[:8] = [[0, 0, 0], [23, 23, 23], [23, 0, 0], [0, 23, 0], [0, 0, 23], [22, 22, 22], [23, 22, 0], [1, 23, 23]]
    xyz = g.origin.astype(np.float64) + g.spacing * idx
    for m in range(g.M):
        v = og.trilinear(m, xyz, grad=False)
        want = g.maps[m, idx[:, 2], idx[:, 1], idx[:, 0]].astype(np.float64)
        assert np.array_equal(v, want)                      # bit-for-bit the stored value


def test_trilinear_exact_on_affine_fields(W, orc):
    T = 3
    coef = [[1.5, -2.0, 0.25, 3.0], [0.0, 0.0, 7.0, -1.0], [-4.0, 0.5, 0.0, 0.0], [2.0, 2.0, 2.0, 2.0], [0.125, -0.75, 1.0, 5.0]]
    g = W.make_affine_grids(12, T, coef)
    og = orc.Grids.from_workload(g)
    rng = np.random.default_rng(1)
    u = rng.uniform(0, 11, (300, 3))
    xyz = u * g.spacing
    for m, (a, b, c, d) in enumerate(coef):
        v, gr = og.trilinear(m, xyz)
        assert np.allclose(v, a * u[:, 0] + b * u[:, 1] + c * u[:, 2] + d, rtol=0, atol=1e-12)
        assert np.allclose(gr, np.array([a, b, c]) / g.spacing, rtol=0, atol=1e-11)


def test_trilinear_matches_library_map_coordinates(tiny):
    g, og = tiny["grids"], tiny["og"]
    rng = np.random.default_rng(2)
    u = rng.uniform(0, 23, (500, 3))                      # (ux,uy,uz) in grid units
    xyz = g.origin.astype(np.float64) + g.spacing * u
    for m in (0, g.M - 2, g.M - 1):
        v = og.trilinear(m, xyz, grad=False)
        want = map_coordinates(g.maps[m].astype(np.float64), [u[:, 2], u[:, 1], u[:, 0]], order=1)
        assert np.allclose(v, want, rtol=1e-12, atol=1e-9)


def test_trilinear_gradient_vs_central_difference(tiny):
    g, og = tiny["grids"], tiny["og"]
    rng = np.random.default_rng(3)
    u = rng.integers(0, 23, (200, 3)) + rng.uniform(0.05, 0.95, (200, 3))
    xyz = g.origin.astype(np.float64) + g.spacing * u
    eps = 1e-3 * g.spacing
    m = g.M - 2                                            # electrostatic map: smooth, O(1) values
    _, gr = og.trilinear(m, xyz)
    for d in range(3):
        e = np.zeros(3); e[d] = eps
        fd = (og.trilinear(m, xyz + e, grad=False) - og.trilinear(m, xyz - e, grad=False)) / (2 * eps)
        assert np.allclose(gr[:, d], fd, rtol=1e-7, atol=1e-7)


def test_grid_atom_weights_and_wall(tiny, par, orc, W):
    g, og = tiny["grids"], tiny["og"]
    T = g.M - 2
    x = g.origin.astype(np.float64) + g.spacing * np.array([5.3, 7.7, 11.2])
    vt, gt = og.trilinear(1, x)
    ve, ge = og.trilinear(T, x)
    vd, gd = og.trilinear(T + 1, x)
    for q in (0.37, -0.37):
        E, gr = og.grid_atom(par, 1, q, T, x)
        assert math.isclose(E, vt[0] + q * ve[0] + abs(q) * vd[0], rel_tol=1e-14)
        assert np.allclose(gr, gt[0] + q * ge[0] + abs(q) * gd[0], rtol=1e-14)
    # outside the box: value of the clamped point + k_wall * distance, gradient k_wall*sign on that axis
    hi = g.box_hi
    for axis, sign, dist in ((0, +1, 0.8), (2, -1, 2.5), (1, +1, 1e-3)):
        xo = x.copy()
        xo[axis] = (hi[axis] + dist) if sign > 0 else (g.box_lo[axis] - dist)
        xc = xo.copy(); xc[axis] = hi[axis] if sign > 0 else g.box_lo[axis]
        Eo, go = og.grid_atom(par, 1, 0.2, T, xo)
        Ec, gc = og.grid_atom(par, 1, 0.2, T, xc)
        assert math.isclose(Eo, Ec + par.k_wall * dist, rel_tol=1e-9)
        assert math.isclose(go[axis], sign * par.k_wall)
        other = [a for a in range(3) if a != axis]
        assert np.allclose(go[other], gc[other], rtol=1e-12)
    # continuity across the face
    xin = x.copy(); xin[0] = hi[0] - 1e-9
    xout = x.copy(); xout[0] = hi[0] + 1e-9
    assert abs(og.grid_atom(par, 1, 0.2, T, xin)[0] - og.grid_atom(par, 1, 0.2, T, xout)[0]) < 1e-3


# ------------------------------------------------------------------------------- R5 pair term
def _zero_grids(orc, c, n=96):
    """all-zero maps on a box wide enough that no atom ever touches the wall"""
    g = c["grids"]
    centre = 0.5 * (g.box_lo + g.box_hi)
    origin = centre - 0.5 * (n - 1) * g.spacing
    return orc.Grids(np.zeros((g.M, n, n, n), np.float32), g.spacing, origin)


def _par_with(orc, W, **kw):
    d = dict(W.DEFAULT_PARAMS); d.update(kw)
    return orc.params(d)


def test_two_atom_closed_forms(orc, W, par):
    Wv, eps, Rm = 0.1662, 0.21, 3.8
    c12, c6 = Wv * eps * Rm ** 12, Wv * 2 * eps * Rm ** 6
    E, dE = orc.pair_energy(par, c12, c6, 6.0, 0.0, 0.0, Rm)
    assert math.isclose(E, -Wv * eps, rel_tol=1e-12) and abs(dE) < 1e-12          # 12-6 minimum
    Wh, eh, Rh = 0.1209, 5.0, 1.9
    c12h, c10 = Wh * 5 * eh * Rh ** 12, Wh * 6 * eh * Rh ** 10
    E, dE = orc.pair_energy(par, c12h, c10, 10.0, 0.0, 0.0, Rh)
    assert math.isclose(E, -Wh * eh, rel_tol=1e-12) and abs(dE) < 1e-10           # 12-10 minimum
    # screened Coulomb: eps(r->inf) -> A+B = 78.4 ; eps(0) = A + B/(1+k)
    p0 = _par_with(orc, W, r_min=1e-12)
    E, _ = orc.pair_energy(p0, 0, 0, 6.0, 0.3, 0.0, 5e3)
    assert math.isclose(E * 5e3, p0.elec_scale * 0.3 / 78.4, rel_tol=1e-6)
    E, _ = orc.pair_energy(p0, 0, 0, 6.0, 0.3, 0.0, 1e-9)
    assert math.isclose(E * 1e-9, p0.elec_scale * 0.3 / (p0.diel_A + p0.diel_B / (1 + p0.diel_k)), rel_tol=1e-6)
    # desolvation: at r=0 equals w_desolv * (S_i V_j + S_j V_i); one sigma out it is e^-1/2 of that
    E0, _ = orc.pair_energy(p0, 0, 0, 6.0, 0.0, 2.5, 0.0)
    assert math.isclose(E0, p0.w_desolv * 2.5, rel_tol=1e-12)
    E1, _ = orc.pair_energy(p0, 0, 0, 6.0, 0.0, 2.5, p0.ds_sigma)
    assert math.isclose(E1, p0.w_desolv * 2.5 * math.exp(-0.5), rel_tol=1e-12)


def test_dielectric_rate_mid_range_closed_forms(orc, W):
    """eps(r) = A + B/(1 + k exp(-lambda*B*r)) (R5): the limits r -> 0 and r -> inf above do not see the RATE
    lambda*B of the sigmoid (lambda*r instead would pass them).  Two hand-worked mid-range points do:
    r = 1/(lambda*B): exp(-1), eps = A + B/(1 + k/e);  r = ln(k)/(lambda*B): k exp(.) = 1, eps = A + B/2."""
    p0 = _par_with(orc, W, r_min=1e-12)
    A, B, k, lam = p0.diel_A, p0.diel_B, p0.diel_k, p0.diel_lambda
    r1 = 1.0 / (lam * B)
    E, _ = orc.pair_energy(p0, 0, 0, 6.0, -0.25, 0.0, r1)
    assert math.isclose(E, p0.elec_scale * -0.25 / ((A + B / (1.0 + k / math.e)) * r1), rel_tol=1e-12)
    r2 = math.log(k) / (lam * B)
    E, _ = orc.pair_energy(p0, 0, 0, 6.0, 0.4, 0.0, r2)
    assert math.isclose(E, p0.elec_scale * 0.4 / ((A + 0.5 * B) * r2), rel_tol=1e-12)
    # the rate is lambda*B = 0.3154 per Angstrom with the literature constants: both points are a few Angstrom out
    assert 3.0 < r1 < 3.3 and 6.0 < r2 < 7.0
    # a wrong rate (lambda alone in the exponent) gives eps(r1) = 1.45 instead of 13.95: the pin is sharp
    E1, _ = orc.pair_energy(p0, 0, 0, 6.0, -0.25, 0.0, r1)
    wrong = p0.elec_scale * -0.25 / ((A + B / (1.0 + k * math.exp(-lam * r1))) * r1)
    assert abs(wrong / E1) > 9.0


def test_pair_derivative_vs_central_difference_and_rmin(orc, par):
    for expA, cA in ((6.0, 800.0), (10.0, 9000.0)):
        for r in (0.9, 1.7, 3.3, 6.0, 11.0):
            E, dE = orc.pair_energy(par, 2.0e5, cA, expA, -0.12, 0.8, r)
            h = 1e-5
            fd = (orc.pair_energy(par, 2.0e5, cA, expA, -0.12, 0.8, r + h)[0] -
                  orc.pair_energy(par, 2.0e5, cA, expA, -0.12, 0.8, r - h)[0]) / (2 * h)
            assert math.isclose(dE, fd, rel_tol=1e-6, abs_tol=1e-9)
    E_in, dE_in = orc.pair_energy(par, 2.0e5, 800.0, 6.0, 0.1, 0.8, 0.2)          # inside r_min: floored, no force
    E_at, _ = orc.pair_energy(par, 2.0e5, 800.0, 6.0, 0.1, 0.8, par.r_min)
    assert E_in == E_at and dE_in == 0.0


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_intra_equals_brute_force_over_all_pairs(cfg, request, orc, par):
    """O(N^2) loop with an on-the-fly exclusion test (library shortest paths + numeric rigidity)."""
    c = request.getfixturevalue(cfg)
    lig, ol, og = c["lig"], c["ol"], c["og"]
    N = lig.N
    A = np.zeros((N, N)); A[lig.bonds[:, 0], lig.bonds[:, 1]] = 1
    D = shortest_path(csr_matrix(A), method="FW", directed=False, unweighted=True)
    rng = np.random.default_rng(9)
    base = ol.pose(ol.identity_genotype())
    d0 = np.linalg.norm(base[:, None] - base[None], axis=-1)
    flex = np.zeros((N, N), bool)
    for _ in range(6):
        g = ol.identity_genotype(); g[7:] = rng.uniform(-3, 3, ol.R)
        x = ol.pose(g)
        flex |= np.abs(np.linalg.norm(x[:, None] - x[None], axis=-1) - d0) > 1e-9
    q = lig.charge.astype(np.float64)
    for trial in range(3):
        g = ol.identity_genotype(); g[7:] = rng.uniform(-3, 3, ol.R)
        g32 = g.astype(np.float32)
        x = ol.pose(g32.astype(np.float64))
        total = 0.0
        for i in range(N):
            for j in range(i + 1, N):
                if D[i, j] <= 3 or not flex[i, j]:
                    continue
                ti, tj = lig.type[i], lig.type[j]
                c12, cA, expA, _ = lig.pair_coeffs[ti, tj].astype(np.float64)
                Si = float(lig.solpar[ti]) + par.qasp * abs(q[i]); Sj = float(lig.solpar[tj]) + par.qasp * abs(q[j])
                dsco = Si * float(lig.vol[tj]) + Sj * float(lig.vol[ti])
                total += orc.pair_energy(par, c12, cA, expA, q[i] * q[j], dsco, np.linalg.norm(x[i] - x[j]))[0]
        r = orc.score(og, ol, par, g32)
        assert math.isclose(r["terms"][0, 1], total, rel_tol=1e-12, abs_tol=1e-12)
        assert math.isclose(r["E"][0], r["terms"][0, 0] + r["terms"][0, 1], rel_tol=1e-15)


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_intra_invariant_under_rigid_motion(cfg, request, orc, par):
    c = request.getfixturevalue(cfg)
    ol, og = c["ol"], c["og"]
    rng = np.random.default_rng(4)
    g = ol.identity_genotype(); g[7:] = rng.uniform(-3, 3, ol.R)
    ref = None
    for _ in range(6):
        g[0:3] = ol.pivot + rng.uniform(-3, 3, 3)
        q = rng.normal(size=4); g[3:7] = q / np.linalg.norm(q)
        intra = orc.score(og, ol, par, g.astype(np.float32))["terms"][0, 1]
        ref = intra if ref is None else ref
        assert math.isclose(intra, ref, rel_tol=1e-5)        # fp32 genotype rounding only
    # exact statement in fp64: zero maps => E = E_intra, compare through score_f64
    zg = _zero_grids(orc, c)
    vals = []
    for _ in range(5):
        g[0:3] = ol.pivot + rng.uniform(-1, 1, 3)
        q = rng.normal(size=4); g[3:7] = q / np.linalg.norm(q)
        vals.append(orc.score_f64(zg, ol, par, g, want_grad=False)[0])
    assert np.ptp(vals) <= 1e-9 * max(1.0, abs(vals[0]))


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_zero_maps_give_zero_rigid_gradient(cfg, request, orc, par):
    """Newton's third law: intramolecular forces produce no net force or torque."""
    c = request.getfixturevalue(cfg)
    ol = c["ol"]
    zg = _zero_grids(orc, c)
    rng = np.random.default_rng(6)
    for _ in range(4):
        g = ol.identity_genotype(); g[7:] = rng.uniform(-3, 3, ol.R)
        q = rng.normal(size=4); g[3:7] = q / np.linalg.norm(q)
        E, gr = orc.score_f64(zg, ol, par, g)
        scale = max(1.0, np.abs(gr[6:]).max())
        assert np.abs(gr[:6]).max() <= 1e-9 * scale
        assert np.abs(gr[6:]).max() > 0


def test_affine_field_translational_gradient(W, orc, par):
    lig = W.make_ligand(12, 3, 3, seed=21, centre=(7.3, 7.3, 7.3))
    lig.charge[:] = 0
    coef = [[1.5, -2.0, 0.25, 3.0], [0.5, 1.0, -1.0, 0.0], [-4.0, 0.5, 2.0, 1.0], [9, 9, 9, 9], [7, 7, 7, 7]]
    g = W.make_affine_grids(40, 3, coef)
    og, ol = orc.Grids.from_workload(g), orc.Ligand.from_workload(lig)
    zero_pairs = lig.pair_coeffs * 0
    ol0 = orc.Ligand(lig.xyz, lig.type, lig.charge, lig.bonds, lig.rot_bonds, 0, 3, zero_pairs, lig.solpar * 0, lig.vol)
    want = sum(np.array(coef[t][:3]) for t in lig.type) / g.spacing
    rng = np.random.default_rng(8)
    for _ in range(4):
        gen = ol0.identity_genotype()
        gen[0:3] += rng.uniform(-0.5, 0.5, 3)
        q = rng.normal(size=4); gen[3:7] = q / np.linalg.norm(q)
        gen[7:] = rng.uniform(-3, 3, ol0.R)
        _, gr = orc.score_f64(og, ol0, par, gen)
        assert np.allclose(gr[:3], want, rtol=1e-10)          # pose independent


# ------------------------------------------------------------------------------- R6 full gradient
def _fd_gradient(orc, og, ol, par, g, eps=1e-5):
    R = ol.R
    fd = np.zeros(6 + R)
    f = lambda gg: orc.score_f64(og, ol, par, gg, want_grad=False)[0]
    for d in range(3):
        e = np.zeros(7 + R); e[d] = eps
        fd[d] = (f(g + e) - f(g - e)) / (2 * eps)
    for d in range(3):                                          # q <- exp(+-eps e_d / 2) (x) q
        w = np.zeros(3); w[d] = eps
        fd[3 + d] = (f(orc.apply_step(R, g, np.concatenate([[0, 0, 0], w, np.zeros(R)]))) -
                     f(orc.apply_step(R, g, np.concatenate([[0, 0, 0], -w, np.zeros(R)])))) / (2 * eps)
    for k in range(R):
        e = np.zeros(7 + R); e[7 + k] = eps
        fd[6 + k] = (f(g + e) - f(g - e)) / (2 * eps)
    return fd


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_analytic_gradient_vs_central_finite_differences(cfg, request, orc, par, W):
    c = request.getfixturevalue(cfg)
    ol, og = c["ol"], c["og"]
    G = W.make_genotypes(400, ol.R, c["grids"], seed=77, wall_tail=0.0)
    r = orc.score(og, ol, par, G)
    # poses with every atom well inside its cell and no pair near the r_min kink
    ok = np.flatnonzero((r["margins"][:, 0] > 2e-3) & (r["margins"][:, 1] > 1e-2))[:12]
    assert len(ok) >= 6
    for i in ok:
        g = G[i].astype(np.float64)
        E, gr = orc.score_f64(og, ol, par, g)
        fd = _fd_gradient(orc, og, ol, par, g)
        scale = np.abs(gr).max()
        assert np.allclose(gr, fd, rtol=1e-6, atol=1e-7 * scale), (i, gr, fd)


def test_gradient_outside_the_box_vs_fd(tiny, orc, par):
    ol, og, grids = tiny["ol"], tiny["og"], tiny["grids"]
    g = ol.identity_genotype()
    g[0] = grids.box_hi[0] + 1.234                            # most atoms beyond the +x face
    g[7:] = [0.4, -0.9]
    E, gr = orc.score_f64(og, ol, par, g)
    fd = _fd_gradient(orc, og, ol, par, g, eps=1e-6)
    assert np.allclose(gr, fd, rtol=1e-5, atol=1e-6 * np.abs(gr).max())
    g[0] = grids.box_hi[0] + 12.0                             # every atom beyond the +x face
    E, gr = orc.score_f64(og, ol, par, g)
    assert math.isclose(gr[0], ol.N * par.k_wall, rel_tol=1e-12)   # the wall pushes back toward the box


def test_degenerate_quaternion_scores_nan(tiny, orc, par):
    g = tiny["ol"].identity_genotype().astype(np.float32)
    g[3:7] = 0
    r = orc.score(tiny["og"], tiny["ol"], par, g)
    assert np.isnan(r["E"][0]) and np.isnan(r["grad"]).all()
