"""CPU (`-m "not gpu"`) checks of the CUDA path's host side: the C-ABI library loads and exports every
symbol include/adock.h declares; its independent ligand preprocessing agrees bit-exactly with the oracle
(R2); the warp-round pair schedule is a conflict-free permutation of the canonical pair list;
error codes for bad arguments.  No compute entry point is called here (no GPU)."""
import ctypes as C
import os
import re
import struct

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2007_03678_b200 import binding
    binding.lib()
    return binding


def test_library_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "adock.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(adock_[a-z_]+)\s*\(", hdr)))
    assert len(declared) >= 16
    L = B.lib()
    for name in declared:
        assert hasattr(L, name), f"libadock.so does not export {name}"
    assert sorted(B.EXPORTS) == declared


def test_default_params_match_the_workload_table(B, W):
    p = B.adock_default_params()
    for k, v in W.DEFAULT_PARAMS.items():
        assert getattr(p, k) == pytest.approx(v, rel=1e-6), k
    assert C.sizeof(B.adock_params) == 18 * 4 + 7 * 4 + 8 * 4     # 18 floats, 7 ints, 8 floats (include/adock.h)


def _host_ligand(B, lig):
    return B.Ligand.from_workload(None, lig)


@pytest.mark.parametrize("name", ["tiny", "mid", "chain", "screen0", "screen1", "screen2", "big"])
def test_integer_structure_bit_exact_vs_oracle(B, W, orc, name, request):
    if name in ("tiny", "mid"):
        lig = request.getfixturevalue(name)["lig"]
    elif name == "chain":
        lig = W.make_chain_ligand(11)
    elif name == "big":
        lig = W.make_ligand(128, 32, 8, seed=3)
    else:
        g = W.make_affine_grids(4, 7, np.zeros((9, 4)))
        lig = W.make_screen_ligands(3, g)[int(name[-1])]
    hl = _host_ligand(B, lig)
    ol = orc.Ligand.from_workload(lig)
    assert np.array_equal(hl.pairs(), ol.pairs)
    t = hl.tree()
    assert np.array_equal(t["tor_order"], ol.tor_order)
    assert np.array_equal(t["moved"], ol.moved)
    assert np.array_equal(t["rot"], ol.rot)
    assert np.array_equal(t["pivot"].astype(np.float64), ol.pivot)


def _parse_image(blob):
    h = struct.unpack_from("18i", blob, 0)
    keys = ["N", "R", "nfrag", "npairs", "nrounds", "T", "off_atoms", "off_meta", "off_frag", "off_fragidx", "off_pairs",
            "bytes", "max_frag_atoms", "max_depth", "npos", "off_fragatoms", "nfull", "systolic"]
    H = dict(zip(keys, h))
    atoms = np.frombuffer(blob, np.float32, 4 * H["npos"], H["off_atoms"]).reshape(-1, 4)
    meta = np.frombuffer(blob, np.uint32, H["npos"], H["off_meta"])
    H["fragatoms"] = np.frombuffer(blob, np.uint16, H["N"], H["off_fragatoms"]).astype(int)
    fg = np.frombuffer(blob, np.float32, 8 * H["nfrag"], H["off_frag"]).reshape(-1, 8)
    fi = np.frombuffer(blob, np.int32, 4 * H["nfrag"], H["off_fragidx"]).reshape(-1, 4)
    pr = np.frombuffer(blob, np.uint32, 4 * 32 * H["nrounds"], H["off_pairs"]).reshape(-1, 32, 4)
    return H, atoms, meta, fg, fi, pr


@pytest.mark.parametrize("name", ["tiny", "mid", "big"])
def test_image_layout_and_conflict_free_schedule(B, W, orc, name, request):
    lig = W.make_ligand(128, 32, 8, seed=3) if name == "big" else request.getfixturevalue(name)["lig"]
    hl = _host_ligand(B, lig)
    ol = orc.Ligand.from_workload(lig)
    blob, int_of_ext = hl.image()
    H, atoms, meta, fg, fi, pr = _parse_image(blob)
    assert (H["N"], H["R"], H["nfrag"], H["npairs"], H["bytes"]) == (lig.N, lig.R, ol.nfrag, ol.npairs, len(blob))
    npos = H["npos"]
    assert npos == 32 * ((lig.N + 31) // 32) and len(set(int_of_ext.tolist())) == lig.N and int_of_ext.max() < npos
    ext_of_int = np.full(npos, -1)
    ext_of_int[int_of_ext] = np.arange(lig.N)
    holes = ext_of_int < 0
    assert (meta[holes] == 0xFFFFFFFF).all() and (meta[~holes] != 0xFFFFFFFF).all()
    occ = np.flatnonzero(~holes)
    # atoms by position: coordinates relative to the pivot, charge, type, fragment id
    piv = hl.tree()["pivot"].astype(np.float64)
    assert np.allclose(atoms[occ, :3], lig.xyz[ext_of_int[occ]].astype(np.float64) - piv, atol=1e-6)
    assert np.array_equal(atoms[occ, 3], lig.charge[ext_of_int[occ]])
    # low byte = cell set of the grid lookup: 2 * type + (charge < 0)   (include/adock.h, adock_load_grids)
    e_occ = ext_of_int[occ]
    assert np.array_equal(meta[occ] & 0xFF, (2 * lig.type[e_occ] + (lig.charge[e_occ] < 0)).astype(np.uint32))
    frag = np.full(npos, -1)
    frag[occ] = (meta[occ] >> 8).astype(int)
    assert sorted(H["fragatoms"].tolist()) == sorted(occ.tolist())
    for f in range(H["nfrag"]):
        parent, a0, a1, w = fi[f]
        members = H["fragatoms"][a0:a1]
        assert (frag[members] == f).all() and (a1 - a0) == (frag == f).sum()
        sub_end, tor = w & 0xFFFF, (w >> 16) & 0xFFFF
        assert f < sub_end <= H["nfrag"]
        if f == 0:
            assert parent == -1 and tor == 0xFFFF and sub_end == H["nfrag"]
        else:
            assert 0 <= parent < f and tor < lig.R
            # the subtree's atoms are exactly the torsion's moved set (canonical numbering)
            sub_atoms = ext_of_int[np.flatnonzero(np.isin(frag, range(f, sub_end)))]
            assert sorted(sub_atoms.tolist()) == np.flatnonzero(ol.moved[tor]).tolist()
            a, b = ol.rot[tor]
            u = lig.xyz[b].astype(np.float64) - lig.xyz[a].astype(np.float64)
            assert np.allclose(fg[f, 4:7], u / np.linalg.norm(u), atol=1e-6)
            assert np.allclose(fg[f, 0:3], lig.xyz[a].astype(np.float64) - piv, atol=1e-6)
    # schedule: a permutation of the canonical pair list, every atom at most once per side per round (hard rule);
    # positions on one side distinct modulo 32 (soft rule, bank-conflict free) in nearly every round.
    # Ligands of exactly four position blocks get the systolic schedule (topology.hpp): round 4 k + b pairs position
    # i = 32 b + lane with j = (i + k + 1) mod npos; excluded pairs are slots with the valid bit clear and zero coefficients.
    assert H["systolic"] == (1 if npos == 128 else 0)
    if H["systolic"]:
        assert H["nrounds"] == (npos // 2) * (npos // 32) and H["nfull"] == 0
        for r in range(H["nrounds"]):
            k, b = divmod(r, npos // 32)
            i = 32 * b + np.arange(32)
            j = (i + k + 1) % npos
            ij = pr[r, :, 0]
            assert np.array_equal(ij & 0x7FF, (i >> 5) * 256 + (i & 31)) and np.array_equal((ij >> 11) & 0x7FF, (j >> 5) * 256 + (j & 31))
            valid = ((ij >> 23) & 1).astype(bool)
            assert (pr[r, ~valid, 1:] == 0).all() and ((ij[~valid] >> 22) == 0).all()
            if k + 1 == npos // 2:
                assert not valid[i >= npos // 2].any()
    seen = []
    wavefronts = []
    for r in range(H["nrounds"]):
        ij = pr[r, :, 0]
        valid = ((ij >> 23) & 1).astype(bool)
        si, sj = (ij & 0x7FF)[valid].astype(int), ((ij >> 11) & 0x7FF)[valid].astype(int)     # slot = (a>>5)*256 + (a&31)
        i, j = (si >> 8) * 32 + (si & 31), (sj >> 8) * 32 + (sj & 31)
        assert ((si & 255) < 32).all() and ((sj & 255) < 32).all() and (ext_of_int[i] >= 0).all() and (ext_of_int[j] >= 0).all()
        assert len(set(i.tolist())) == len(i) and len(set(j.tolist())) == len(j)
        if len(i):
            wavefronts += [np.bincount(i & 31).max(), np.bincount(j & 31).max()]      # replays of one 4-byte access
        if not H["systolic"]:
            assert (pr[r, ~valid] == 0).all() and (valid.all() == (r < H["nfull"]))
        for a, b, rec in zip(i, j, pr[r, valid]):
            ea, eb = int(ext_of_int[a]), int(ext_of_int[b])
            seen.append((min(ea, eb), max(ea, eb)))
            c12, cA = np.frombuffer(rec[1:3].tobytes(), np.float32)
            co = lig.pair_coeffs[lig.type[ea], lig.type[eb]]
            assert (c12, cA) == (co[0], co[1]) and int((rec[0] >> 22) & 1) == int(co[2] > 8)
    assert sorted(seen) == [tuple(p) for p in ol.pairs.tolist()]
    # packing efficiency against the lower bound max(ceil(np/32), ceil(max degree / 2))
    deg = np.bincount(ol.pairs.ravel(), minlength=lig.N).max()
    lower = max(int(np.ceil(ol.npairs / 32)), int(np.ceil(deg / 2)))
    assert H["nrounds"] <= int(np.ceil(1.3 * lower)) + 1, (H["nrounds"], lower)
    assert np.mean(wavefronts) <= 2.0 and max(wavefronts) <= 3, (np.mean(wavefronts), max(wavefronts))
    if H["systolic"]:
        assert max(wavefronts) == 1


def test_load_ligand_rejects_bad_input(B, W):
    lig = W.make_chain_ligand(8)
    with pytest.raises(B.AdockError) as e:
        bad = W.make_chain_ligand(8); bad.type[0] = 9
        _host_ligand(B, bad)
    assert e.value.code == B.ADOCK_EINVAL
    with pytest.raises(B.AdockError) as e:
        ring = W.make_chain_ligand(8); ring.bonds = np.concatenate([ring.bonds, [[0, 7]]]).astype(np.int32)
        _host_ligand(B, ring)
    assert e.value.code == B.ADOCK_EINVAL and "ring" in str(e.value)
    with pytest.raises(B.AdockError) as e:
        nb = W.make_chain_ligand(8); nb.rot_bonds = np.array([[0, 5]], np.int32)
        _host_ligand(B, nb)
    assert e.value.code == B.ADOCK_EINVAL
    with pytest.raises(B.AdockError) as e:
        nan = W.make_chain_ligand(8); nan.xyz[3, 1] = np.nan
        _host_ligand(B, nan)
    assert e.value.code == B.ADOCK_EINVAL
    with pytest.raises(B.AdockError) as e:
        big = W.make_chain_ligand(8)
        B.Ligand(None, np.zeros((300, 3), np.float32), np.zeros(300, np.int32), np.zeros(300, np.float32), big.bonds, big.rot_bonds,
                 0, 2, big.pair_coeffs, big.solpar, big.vol)
    assert e.value.code == B.ADOCK_ELIMIT
    assert _host_ligand(B, lig).pairs().shape == (10, 2)


def test_shard_partitions_ligands_without_overlap(W):
    for n, world in ((10, 2), (7, 4), (3, 8)):
        parts = [W.shard(n, r, world) for r in range(world)]
        assert sorted(sum(parts, [])) == list(range(n))
        assert max(map(len, parts)) - min(map(len, parts)) <= 1
