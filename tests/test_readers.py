"""PDBQT and AutoGrid .map readers: round trips of synthetic
ligands and maps through the writers, a hand-written PDBQT fragment, and the error cases.  The decisive check: the
ligand read back has the same integer structure (pairs, fragments, torsion tree) in the oracle as the original."""
import numpy as np
import pytest

from paper_2007_03678_b200 import readers as RD

NAMES = ["C", "A", "N", "NA", "OA", "HD", "S"]


@pytest.mark.parametrize("seed,N,R", [(1, 16, 2), (2, 40, 8), (3, 33, 0), (4, 60, 15)])
def test_pdbqt_round_trip_preserves_structure(W, orc, seed, N, R):
    lig = W.make_ligand(N, R, 7, seed, (12.0, 12.0, 12.0))
    text, order = RD.write_pdbqt(lig, NAMES)
    back = RD.read_pdbqt(text, NAMES, lig.pair_coeffs, lig.solpar, lig.vol)
    order = np.array(order)
    assert back.N == lig.N and back.R == lig.R
    assert np.abs(back.xyz - lig.xyz[order]).max() <= 5.1e-4               # %8.3f
    assert np.abs(back.charge - lig.charge[order]).max() <= 5.1e-4
    assert np.array_equal(back.type, lig.type[order])
    inv = np.empty(N, int); inv[order] = np.arange(N)
    as_set = lambda b, m=None: {tuple(sorted((int(x), int(y)))) for x, y in (b if m is None else m[b])}
    assert as_set(back.bonds) == as_set(lig.bonds, inv)
    assert as_set(back.rot_bonds) == as_set(lig.rot_bonds, inv)
    assert back.root_atom == inv[lig.root_atom] == 0
    # same non-excluded pair set and fragment partition in the oracle, up to the renumbering
    a, b = orc.Ligand.from_workload(lig), orc.Ligand.from_workload(back)
    assert as_set(b.pairs) == as_set(a.pairs, inv)
    assert b.nfrag == a.nfrag and sorted(np.bincount(b.frag).tolist()) == sorted(np.bincount(a.frag).tolist())


def test_pdbqt_hand_written_and_bond_inference():
    text = """REMARK  a 4-atom chain C-C-O-H with one rotatable bond, no CONECT records
ROOT
ATOM      1  C1  LIG A   1       0.000   0.000   0.000  1.00  0.00     0.100 C 
ATOM      2  C2  LIG A   1       1.500   0.000   0.000  1.00  0.00    -0.050 C 
ENDROOT
BRANCH   2   3
ATOM      3  O1  LIG A   1       2.200   1.200   0.000  1.00  0.00    -0.400 OA
ATOM      4  H1  LIG A   1       3.150   1.100   0.000  1.00  0.00     0.350 HD
ENDBRANCH   2   3
TORSDOF 1
"""
    T = len(NAMES)
    lig = RD.read_pdbqt(text, NAMES, np.zeros((T, T, 4)), np.zeros(T), np.zeros(T))
    assert lig.N == 4 and lig.R == 1 and lig.root_atom == 0
    assert lig.type.tolist() == [0, 0, 4, 5]
    assert np.allclose(lig.charge, [0.1, -0.05, -0.4, 0.35])
    assert np.allclose(lig.xyz[2], [2.2, 1.2, 0.0])
    assert lig.rot_bonds.tolist() == [[1, 2]]
    assert lig.bonds.tolist() == [[0, 1], [1, 2], [2, 3]]                  # inferred from distances + the BRANCH bond
    with pytest.raises(ValueError, match="no map"):
        RD.read_pdbqt(text.replace(" OA", " ZN"), NAMES, np.zeros((T, T, 4)), np.zeros(T), np.zeros(T))
    with pytest.raises(ValueError, match="unknown atom serial"):
        RD.read_pdbqt(text.replace("BRANCH   2   3", "BRANCH   2   9"), NAMES, np.zeros((T, T, 4)), np.zeros(T), np.zeros(T))
    with pytest.raises(ValueError, match="no ATOM"):
        RD.read_pdbqt("ROOT\nENDROOT\n", NAMES, np.zeros((T, T, 4)), np.zeros(T), np.zeros(T))


def test_map_round_trip_and_geometry(W):
    grids, _ = W.make_config("tiny")
    texts = [RD.write_map(m, grids.spacing, grids.origin) for m in grids.maps]
    back = RD.read_maps(texts)
    assert back.maps.shape == grids.maps.shape and back.dims == grids.dims
    assert np.array_equal(back.maps, grids.maps)                           # %.9g round-trips float32 exactly
    assert back.spacing == pytest.approx(grids.spacing) and np.allclose(back.origin, grids.origin, atol=1e-5)
    # x fastest: value k of the file is node (k % nx, (k // nx) % ny, k // (nx ny))
    nx, ny, nz = grids.dims
    vals = [float(v) for v in texts[0].splitlines()[6:]]
    assert vals[1] == grids.maps[0, 0, 0, 1] and vals[nx] == grids.maps[0, 0, 1, 0] and vals[nx * ny] == grids.maps[0, 1, 0, 0]
    with pytest.raises(ValueError, match="differ"):
        RD.read_maps([texts[0], texts[1].replace("SPACING 0.375000", "SPACING 0.400000")])
    with pytest.raises(ValueError, match="values"):
        RD.read_maps(["\n".join(texts[0].splitlines()[:-5]) + "\n"])
    with pytest.raises(ValueError, match="header"):
        RD.read_maps([texts[0].replace("SPACING", "SPACE")])


# ------------------------------------------------------------------- hand-typed files in the public layouts (tests/golden)
def _golden(name):
    import os
    return open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)).read()


def test_hand_typed_pdbqt_in_the_public_column_layout(orc):
    """tests/golden/toy_ligand.pdbqt was typed by hand against the public PDBQT layout (PDB fixed columns: serial 7-11,
    x 31-38, y 39-46, z 47-54, partial charge 71-76, AutoDock atom type 78-79; ROOT / ENDROOT, nested BRANCH a b /
    ENDBRANCH a b, TORSDOF), not produced by write_pdbqt: a column mistake shared by reader and writer fails here.
    Expected arrays typed independently below."""
    text = _golden("toy_ligand.pdbqt")
    # the columns, checked without the reader: atom 4 (file line 8)
    ln = text.splitlines()[7]
    assert ln[0:6] == "ATOM  " and ln[6:11] == "    4" and ln[30:38] == "   2.250" and ln[38:46] == "   1.299" and ln[46:54] == "   0.000"
    assert ln[70:76] == "-0.350" and ln[77:79] == "OA"
    names = ["C", "N", "OA", "HD"]
    T = len(names)
    lig = RD.read_pdbqt(text, names, np.zeros((T, T, 4), np.float32) + np.array([1, 1, 6, 0], np.float32), np.zeros(T), np.ones(T))
    xyz = np.array([[0, 0, 0], [1.5, 0, 0], [-0.75, 1.299, 0], [2.25, 1.299, 0], [3.75, 1.299, 0], [4.5, 2.598, 0], [5.58, 2.598, 0],
                    [-2.25, 1.299, 0]], np.float32)
    assert lig.N == 8 and np.array_equal(lig.xyz, xyz)
    assert np.array_equal(lig.charge, np.array([0.05, -0.02, -0.3, -0.35, 0.12, 0.01, 0.2, 0.09], np.float32))
    assert lig.type.tolist() == [0, 0, 1, 2, 0, 0, 3, 0]
    assert lig.root_atom == 0 and lig.R == 3
    assert sorted(map(tuple, lig.rot_bonds.tolist())) == [(1, 3), (2, 7), (4, 5)]          # BRANCH serials 2-4, 3-8, 5-6
    # no CONECT records: bonds from the distance rule (1.5 A heavy-atom bonds, 1.08 A C-H) plus the BRANCH bonds
    assert sorted(map(tuple, lig.bonds.tolist())) == [(0, 1), (0, 2), (1, 3), (2, 7), (3, 4), (4, 5), (5, 6)]
    # the oracle's preprocessing (R2) on it: 4 rigid fragments {0,1,2}, {3,4}, {5,6}, {7}; torsion 5-6 is nested in 2-4
    ol = orc.Ligand.from_workload(lig)
    assert ol.nfrag == 4 and ol.frag.tolist() == [0, 0, 0, 1, 1, 2, 2, 3]
    moved = {(int(a), int(b)): ol.moved[k].nonzero()[0].tolist() for k, (a, b) in enumerate(ol.rot)}
    assert moved == {(1, 3): [3, 4, 5, 6], (4, 5): [5, 6], (2, 7): [7]}


def test_hand_typed_autogrid_map_in_the_public_layout():
    """tests/golden/toy.C.map: six header lines (GRID_PARAMETER_FILE, GRID_DATA_FILE, MACROMOLECULE, SPACING, NELEMENTS =
    numbers of INTERVALS, CENTER), then one value per line with x fastest, then y, then z; value = ix + 10 iy + 100 iz + 0.5."""
    text = _golden("toy.C.map")
    g = RD.read_maps([text, text, text])
    assert g.maps.shape == (3, 3, 3, 3) and g.spacing == 0.375
    assert np.allclose(g.origin, [1.0 - 0.375, 2.0 - 0.375, 3.0 - 0.375])                  # CENTER - spacing * NELEMENTS / 2
    iz, iy, ix = np.meshgrid(np.arange(3), np.arange(3), np.arange(3), indexing="ij")
    assert np.array_equal(g.maps[0], (ix + 10 * iy + 100 * iz + 0.5).astype(np.float32))    # [z][y][x]
    assert g.maps[0][2, 1, 0] == 210.5 and g.maps[0][0, 1, 2] == 12.5
