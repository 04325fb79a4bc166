"""Pins for the oracle's ligand preprocessing (R2) and pose builder (R3).

PAPER.md lines 58/110 only name "ligand pose" and "torsions"; the pins are what geometry fixes:
identity pose, rigid-body invariants, hand-countable chains, brute-force rigidity, library
shortest paths and library rotations.
"""
import math

import numpy as np
import pytest
from scipy.sparse import csr_matrix
from scipy.sparse.csgraph import shortest_path
from scipy.spatial.transform import Rotation


def _rand_geno(rng, R, centre, spread=2.0):
    g = np.zeros(7 + R)
    g[0:3] = centre + rng.uniform(-spread, spread, 3)
    q = rng.normal(size=4)
    g[3:7] = q / np.linalg.norm(q)
    g[7:] = rng.uniform(-math.pi, math.pi, R)
    return g


@pytest.mark.parametrize("N", [6, 9, 14])
def test_chain_closed_forms(W, orc, N):
    lig = W.make_chain_ligand(N)
    ol = orc.Ligand.from_workload(lig)
    R = N - 3
    assert ol.R == R and ol.nfrag == R + 1
    # bond k=(k,k+1), k=1..N-3 (torsion index k-1): moved set = atoms k+1..N-1, depth = k
    for t in range(R):
        k = t + 1
        assert ol.rot[t].tolist() == [k, k + 1]
        assert ol.moved[t].tolist() == [0] * (k + 1) + [1] * (N - 1 - k)
        assert ol.depth[t] == k
    assert ol.moved.sum() == sum(N - 1 - k for k in range(1, N - 2))
    assert ol.tor_order.tolist() == list(range(R - 1, -1, -1))          # deepest first
    # every pair with |i-j| >= 4 is flexible and non-excluded: (N-4)(N-3)/2 of them, lexicographic
    want = [(i, j) for i in range(N) for j in range(i + 1, N) if j - i >= 4]
    assert ol.npairs == (N - 4) * (N - 3) // 2 == len(want)
    assert ol.pairs.tolist() == [list(p) for p in want]


def test_reversed_rot_bond_is_reoriented(W, orc):
    lig = W.make_chain_ligand(8)
    lig.rot_bonds = lig.rot_bonds[:, ::-1].copy()
    ol = orc.Ligand.from_workload(lig)
    assert (ol.rot[:, 0] < ol.rot[:, 1]).all()


def test_ring_bond_rejected(W, orc):
    lig = W.make_chain_ligand(8)
    lig.bonds = np.concatenate([lig.bonds, np.array([[0, 7]], np.int32)])   # closes a ring over all bonds
    with pytest.raises(ValueError):
        orc.Ligand.from_workload(lig)


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_bfs_vs_library_shortest_path(cfg, request):
    c = request.getfixturevalue(cfg)
    lig, ol = c["lig"], c["ol"]
    N = lig.N
    A = np.zeros((N, N))
    A[lig.bonds[:, 0], lig.bonds[:, 1]] = 1
    D = shortest_path(csr_matrix(A), method="FW", directed=False, unweighted=True)
    assert (ol.dist == D.astype(np.int32)).all()


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_pair_list_vs_brute_force_rigidity(cfg, request):
    """pair (i<j) is listed  <=>  d(i,j) > 3 and |x_i-x_j| changes under some random torsion setting."""
    c = request.getfixturevalue(cfg)
    lig, ol = c["lig"], c["ol"]
    rng = np.random.default_rng(5)
    base = ol.pose(ol.identity_genotype())
    d0 = np.linalg.norm(base[:, None] - base[None], axis=-1)
    changed = np.zeros_like(d0, bool)
    for _ in range(6):
        g = ol.identity_genotype()
        g[7:] = rng.uniform(-math.pi, math.pi, ol.R)
        x = ol.pose(g)
        d = np.linalg.norm(x[:, None] - x[None], axis=-1)
        changed |= np.abs(d - d0) > 1e-9
    want = [[i, j] for i in range(lig.N) for j in range(i + 1, lig.N) if ol.dist[i, j] > 3 and changed[i, j]]
    assert ol.pairs.tolist() == want
    assert 0 < ol.npairs <= lig.N * (lig.N - 1) // 2


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_fragments_and_depths(cfg, request):
    c = request.getfixturevalue(cfg)
    lig, ol = c["lig"], c["ol"]
    assert ol.nfrag == ol.R + 1                      # tree: each rotatable bond splits one fragment
    assert ol.frag[0] == 0 and (np.diff(np.unique(ol.frag)) == 1).all()
    for k in range(ol.R):
        a, b = ol.rot[k]
        assert ol.moved[k, b] == 1 and ol.moved[k, a] == 0 and ol.moved[k, lig.root_atom] == 0
        assert ol.depth[k] >= 1
        assert ol.depth[k] == sum(int(ol.moved[k2, b]) for k2 in range(ol.R))
    d = ol.depth[ol.tor_order]
    assert (np.diff(d) <= 0).all()
    # pivot = mean of input coordinates, rounded once to fp32
    assert np.array_equal(ol.pivot, lig.xyz.astype(np.float64).mean(0).astype(np.float32).astype(np.float64))


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_identity_genotype_reproduces_input(cfg, request):
    c = request.getfixturevalue(cfg)
    x = c["ol"].pose(c["ol"].identity_genotype())
    assert np.abs(x - c["lig"].xyz.astype(np.float64)).max() <= 1e-12


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_rigid_invariants_under_random_genotypes(cfg, request):
    c = request.getfixturevalue(cfg)
    lig, ol = c["lig"], c["ol"]
    rng = np.random.default_rng(11)
    x0 = lig.xyz.astype(np.float64)
    d0 = np.linalg.norm(x0[:, None] - x0[None], axis=-1)
    same_frag = ol.frag[:, None] == ol.frag[None]
    for _ in range(8):
        g = _rand_geno(rng, ol.R, ol.pivot)
        x = ol.pose(g)
        d = np.linalg.norm(x[:, None] - x[None], axis=-1)
        assert np.abs(d - d0)[same_frag].max() < 1e-10                       # fragments stay rigid
        bl = d[lig.bonds[:, 0], lig.bonds[:, 1]]
        assert np.abs(bl - 1.5).max() < 1e-5                                 # every bond length kept
        g2 = g.copy(); g2[7:] += 2 * math.pi
        assert np.abs(ol.pose(g2) - x).max() < 1e-9                          # tau periodic
        g3 = g.copy(); g3[3:7] *= -1
        assert np.abs(ol.pose(g3) - x).max() < 1e-12                         # q and -q
        g4 = g.copy(); g4[3:7] *= 3.7
        assert np.abs(ol.pose(g4) - x).max() < 1e-12                         # normalised on use
        g5 = g.copy(); g5[0:3] += [0.3, -1.1, 2.0]
        assert np.abs(ol.pose(g5) - (x + [0.3, -1.1, 2.0])).max() < 1e-12    # pure translation


def test_quaternion_matches_library_rotation(tiny):
    ol = tiny["ol"]
    rng = np.random.default_rng(3)
    x0 = ol.pose(ol.identity_genotype())
    for _ in range(5):
        g = ol.identity_genotype()
        q = rng.normal(size=4); q /= np.linalg.norm(q)
        g[3:7] = q
        g[0:3] = [1.0, 2.0, 3.0]
        want = Rotation.from_quat([q[1], q[2], q[3], q[0]]).apply(x0 - ol.pivot) + g[0:3]   # scipy order x,y,z,w
        assert np.abs(ol.pose(g) - want).max() < 1e-12
    # textbook quarter turn about z: (x,y,z) -> (-y,x,z)
    g = ol.identity_genotype()
    g[3:7] = [math.sqrt(0.5), 0, 0, math.sqrt(0.5)]
    v = x0 - ol.pivot
    assert np.abs(ol.pose(g) - (np.stack([-v[:, 1], v[:, 0], v[:, 2]], 1) + ol.pivot)).max() < 1e-12
    with pytest.raises(ValueError):
        g[3:7] = 0
        ol.pose(g)


@pytest.mark.parametrize("cfg", ["tiny", "mid"])
def test_single_torsion_is_right_handed_rotation_about_axis(cfg, request):
    c = request.getfixturevalue(cfg)
    lig, ol = c["lig"], c["ol"]
    x0 = lig.xyz.astype(np.float64)
    for k in range(ol.R):
        a, b = ol.rot[k]
        u = (x0[b] - x0[a]) / np.linalg.norm(x0[b] - x0[a])
        for tau in (0.7, -2.1):
            g = ol.identity_genotype()
            g[7 + k] = tau
            x = ol.pose(g)
            mv = ol.moved[k].astype(bool)
            assert np.abs(x[~mv] - x0[~mv]).max() < 1e-12
            want = Rotation.from_rotvec(tau * u).apply(x0[mv] - x0[a]) + x0[a]          # library Rodrigues
            assert np.abs(x[mv] - want).max() < 1e-10


def test_nested_torsions_compose_root_to_leaf(mid):
    """deepest-first in the reference frame == rotating the posed subtree about the posed axis."""
    ol, lig = mid["ol"], mid["lig"]
    x0 = lig.xyz.astype(np.float64)
    # find a nested pair: k2 deeper than k1 and b_k2 in M_k1
    for k1 in range(ol.R):
        for k2 in range(ol.R):
            if k1 != k2 and ol.moved[k1, ol.rot[k2][1]] and ol.moved[k1, ol.rot[k2][0]]:
                g = ol.identity_genotype()
                g[7 + k1], g[7 + k2] = 0.9, -1.3
                x = ol.pose(g)
                a1, b1 = ol.rot[k1]
                u1 = (x0[b1] - x0[a1]) / np.linalg.norm(x0[b1] - x0[a1])
                R1 = Rotation.from_rotvec(0.9 * u1)
                y = x0.copy()
                m1 = ol.moved[k1].astype(bool)
                y[m1] = R1.apply(x0[m1] - x0[a1]) + x0[a1]          # shallow torsion first ...
                a2, b2 = ol.rot[k2]
                u2 = (y[b2] - y[a2]) / np.linalg.norm(y[b2] - y[a2])  # ... then the deep one about its MOVED axis
                m2 = ol.moved[k2].astype(bool)
                y[m2] = Rotation.from_rotvec(-1.3 * u2).apply(y[m2] - y[a2]) + y[a2]
                assert np.abs(x - y).max() < 1e-10
                return
    pytest.skip("no nested torsions in this ligand")
