"""Pins for the oracle's pose post-processing (R13; RMSD between poses): closed forms of
the RMSD and a hand-worked clustering example."""
import numpy as np


def test_rmsd_closed_forms(orc):
    rng = np.random.default_rng(0)
    x = rng.normal(size=(17, 3))
    assert orc.pose_rmsd(x, x) == 0.0
    t = np.array([0.3, -1.2, 2.0])
    assert np.isclose(orc.pose_rmsd(x + t, x), np.linalg.norm(t), rtol=1e-14)          # rigid shift: |t|
    y = x.copy(); y[5] += [3.0, 4.0, 0.0]
    assert np.isclose(orc.pose_rmsd(y, x), 5.0 / np.sqrt(17), rtol=1e-14)             # one atom moved by 5
    # rotation by pi about z of points on the x axis: each moves by 2|x|
    p = np.zeros((4, 3)); p[:, 0] = [1, 2, 3, 4]
    assert np.isclose(orc.pose_rmsd(p * [-1, -1, 1], p), 2 * np.sqrt((p[:, 0] ** 2).mean()), rtol=1e-14)
    P = orc.pose_rmsd_pairs(rng.normal(size=(6, 9, 3)))
    assert np.allclose(P, P.T) and np.all(np.diag(P) == 0)
    for i in range(6):
        for j in range(6):
            for k in range(6):
                assert P[i, j] <= P[i, k] + P[k, j] + 1e-12                          # a metric on R^(3N)


def test_clustering_hand_example(orc):
    """one-atom poses on a line at 0, 0.5, 3, 3.4, 10, 2.2; tol 1: by energy order 2 (E=-9) seeds cluster 0, 0 (E=-8)
    seeds cluster 1, 3 joins 0, 1 joins 1, 5 (2.2: 0.8 from pose 2) joins 0, 4 seeds cluster 2."""
    pos = np.array([0.0, 0.5, 3.0, 3.4, 10.0, 2.2])
    x = np.zeros((6, 1, 3)); x[:, 0, 0] = pos
    E = np.array([-8.0, -5.0, -9.0, -7.0, -1.0, -6.0])
    P = orc.pose_rmsd_pairs(x)
    assert np.allclose(P, np.abs(pos[:, None] - pos[None, :]))
    c, n = orc.cluster_poses(E, P, 1.0)
    assert n == 3 and c.tolist() == [1, 1, 0, 0, 2, 0]
    # ties in energy: lower index first
    c2, n2 = orc.cluster_poses(np.zeros(6), P, 1.0)
    assert c2.tolist() == [0, 0, 1, 1, 2, 1] and n2 == 3      # pose 5 (2.2) is 0.8 from seed 2 (3.0)
