"""Thin ctypes binding over the C-ABI library (include/adock.h): argument marshalling only.

Device buffers are torch CUDA tensors (PyTorch is used for device memory and streams, nothing else);
every step of the path runs in the library's CUDA kernels.  There is no CPU fallback: if libadock.so is
missing or CUDA is unavailable, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

ADOCK_OK, ADOCK_EINVAL, ADOCK_ENOMEM, ADOCK_ECUDA, ADOCK_ELIMIT = 0, -1, -2, -3, -4
EXPORTS = ["adock_default_params", "adock_load_grids", "adock_free_grids", "adock_load_ligand", "adock_free_ligand",
           "adock_ligand_pairs", "adock_ligand_tree", "adock_ligand_image", "adock_score_batch", "adock_score_batch_host", "adock_local_search",
           "adock_philox", "adock_ga_generation", "adock_dock", "adock_dock_many", "adock_launch_count", "adock_last_error", "adock_profile", "adock_profile_read",
           "adock_ligand_lane_image", "adock_set_path", "adock_last_dock_path", "adock_solis_wets", "adock_screen", "adock_pose_rmsd", "adock_alu_peak", "adock_tmem_probe", "adock_local_search_noalloc"]


class adock_ligand_desc(C.Structure):
    _fields_ = [("N", C.c_int), ("xyz", C.c_void_p), ("type", C.c_void_p), ("charge", C.c_void_p), ("nbonds", C.c_int),
                ("bonds", C.c_void_p), ("R", C.c_int), ("rot_bonds", C.c_void_p), ("root_atom", C.c_int)]


class adock_screen_stats(C.Structure):
    _fields_ = [("wall_s", C.c_double), ("dock_s", C.c_double), ("prep_s", C.c_double), ("exposed_s", C.c_double),
                ("batches", C.c_int), ("host_threads", C.c_int)]


class AdockError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"adock error {code}: {msg}")
        self.code = code


class adock_params(C.Structure):
    _fields_ = [(k, C.c_float) for k in (
        "elec_scale", "diel_A", "diel_B", "diel_k", "diel_lambda", "w_desolv", "ds_sigma", "qasp", "r_min", "k_wall",
        "ad_rho", "ad_eps", "lsrat", "tourn_prob", "xover_rate", "mut_rate", "dmov", "dang")] + [
        (k, C.c_int) for k in ("lsit", "max_gens", "ls_method", "sw_max_succ", "sw_max_fail", "autostop", "as_window")] + [
        (k, C.c_float) for k in ("sw_rho0", "sw_rho_lb", "sw_expand", "sw_contract", "sw_bias_keep", "sw_bias_gain",
                                 "sw_bias_decay", "as_tol")]


def lib():
    """Load libadock.so (building it when nvcc is present and it is stale). Fails loudly when absent."""
    global _lib
    if _lib is None:
        if _build.stale():
            _build.build()
        if not os.path.exists(_build.LIB):
            raise ImportError("libadock.so is missing: run paper_2007_03678_b200.build.build() (needs nvcc)")
        L = C.CDLL(_build.LIB)
        vp, ci, cf = C.c_void_p, C.c_int, C.c_float
        pp = C.POINTER(adock_params)
        L.adock_last_error.restype = C.c_char_p
        L.adock_launch_count.restype = C.c_longlong
        L.adock_launch_count.argtypes = [ci]
        L.adock_default_params.argtypes = [pp]
        L.adock_load_grids.argtypes = [vp, ci, ci, ci, ci, cf, vp, C.POINTER(vp)]
        L.adock_free_grids.argtypes = [vp]
        L.adock_free_grids.restype = None
        L.adock_load_ligand.argtypes = [vp, pp, ci, vp, vp, vp, ci, vp, ci, vp, ci, ci, vp, vp, vp, C.POINTER(vp)]
        L.adock_free_ligand.argtypes = [vp]
        L.adock_free_ligand.restype = None
        L.adock_ligand_pairs.argtypes = [vp, C.POINTER(ci), C.POINTER(vp)]
        L.adock_ligand_tree.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.adock_ligand_image.argtypes = [vp, C.POINTER(ci), C.POINTER(vp), C.POINTER(vp)]
        L.adock_ligand_lane_image.argtypes = [vp, C.POINTER(ci), C.POINTER(vp), C.POINTER(vp)]
        L.adock_set_path.argtypes = [ci]
        L.adock_score_batch.argtypes = [vp, vp, pp, vp, ci, ci, vp, vp, vp, ci, vp]
        L.adock_score_batch_host.argtypes = [vp, vp, pp, vp, ci, ci, vp, vp, vp, ci, vp]
        L.adock_local_search.argtypes = [vp, vp, pp, vp, ci, ci, vp, vp, vp, vp]
        L.adock_local_search_noalloc.argtypes = [vp, vp, pp, vp, ci, ci, vp, vp, vp, vp]
        L.adock_solis_wets.argtypes = [vp, vp, pp, vp, ci, ci, vp, vp, vp, C.c_ulonglong, C.c_uint, vp]
        L.adock_philox.argtypes = [vp, vp, ci, vp, vp]
        L.adock_ga_generation.argtypes = [vp, vp, pp, ci, ci, ci, C.c_ulonglong, vp, vp, vp, vp, vp, C.POINTER(ci), vp]
        L.adock_dock.argtypes = [vp, vp, pp, ci, ci, C.c_longlong, C.c_ulonglong, vp, vp, vp, vp, vp, vp]
        L.adock_dock_many.argtypes = [vp, vp, ci, pp, ci, ci, C.c_longlong, vp, ci, vp, vp, ci, vp, vp, vp, vp]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise AdockError(rc, lib().adock_last_error().decode())


def _np(a, dt):
    return np.ascontiguousarray(a, dt)


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t):
    """device pointer of a torch CUDA tensor (or None)"""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device buffers must be contiguous CUDA tensors"
    return C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def adock_default_params() -> adock_params:
    p = adock_params()
    _check(lib().adock_default_params(C.byref(p)))
    return p


def make_params(d: dict | None = None) -> adock_params:
    """adock_params from a name->value dict (workloads.DEFAULT_PARAMS style); missing names keep defaults."""
    p = adock_default_params()
    for k, v in (d or {}).items():
        setattr(p, k, v)
    return p


class Grids:
    """adock_load_grids / adock_free_grids"""

    def __init__(self, maps, spacing, origin):
        maps = _np(maps, np.float32)
        assert maps.ndim == 4
        self.M, self.nz, self.ny, self.nx = maps.shape
        self.spacing = float(spacing)
        self.h = C.c_void_p()
        _check(lib().adock_load_grids(_hp(maps), self.M, self.nx, self.ny, self.nz, self.spacing, _hp(_np(origin, np.float32)),
                                      C.byref(self.h)))

    @classmethod
    def from_workload(cls, g):
        return cls(g.maps, g.spacing, g.origin)

    def close(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.adock_free_grids(self.h)
            self.h = None

    __del__ = close


class Ligand:
    """adock_load_ligand / adock_free_ligand / adock_ligand_pairs / adock_ligand_tree"""

    def __init__(self, grids: Grids, xyz, type, charge, bonds, rot_bonds, root_atom, T, pair_coeffs, solpar, vol, params=None):
        xyz, type, charge = _np(xyz, np.float32), _np(type, np.int32), _np(charge, np.float32)
        bonds, rot = _np(bonds, np.int32).reshape(-1, 2), _np(rot_bonds, np.int32).reshape(-1, 2)
        self.N, self.R, self.T = int(xyz.shape[0]), int(rot.shape[0]), int(T)
        self.h = C.c_void_p()
        _check(lib().adock_load_ligand(grids.h if grids is not None else None, C.byref(params) if params is not None else None, self.N, _hp(xyz), _hp(type),
                                       _hp(charge), bonds.shape[0], _hp(bonds), self.R, _hp(rot), int(root_atom), self.T,
                                       _hp(_np(pair_coeffs, np.float32)), _hp(_np(solpar, np.float32)), _hp(_np(vol, np.float32)),
                                       C.byref(self.h)))

    @classmethod
    def from_workload(cls, grids: Grids, lig, params=None):
        return cls(grids, lig.xyz, lig.type, lig.charge, lig.bonds, lig.rot_bonds, lig.root_atom, lig.T, lig.pair_coeffs,
                   lig.solpar, lig.vol, params)

    def pairs(self) -> np.ndarray:
        n, p = C.c_int(), C.c_void_p()
        _check(lib().adock_ligand_pairs(self.h, C.byref(n), C.byref(p)))
        if n.value == 0:
            return np.zeros((0, 2), np.int32)
        return np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_int)), (n.value, 2)).copy()

    def tree(self):
        o, m, r, pv = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(lib().adock_ligand_tree(self.h, C.byref(o), C.byref(m), C.byref(r), C.byref(pv)))
        R, N = self.R, self.N
        order = np.ctypeslib.as_array(C.cast(o, C.POINTER(C.c_int)), (R,)).copy() if R else np.zeros(0, np.int32)
        moved = np.ctypeslib.as_array(C.cast(m, C.POINTER(C.c_ubyte)), (R, N)).copy() if R else np.zeros((0, N), np.uint8)
        rot = np.ctypeslib.as_array(C.cast(r, C.POINTER(C.c_int)), (R, 2)).copy() if R else np.zeros((0, 2), np.int32)
        pivot = np.ctypeslib.as_array(C.cast(pv, C.POINTER(C.c_float)), (3,)).copy()
        return dict(tor_order=order, moved=moved, rot=rot, pivot=pivot)

    def image(self):
        """(host copy of the device image as bytes, int_of_ext [N])"""
        n, p, m = C.c_int(), C.c_void_p(), C.c_void_p()
        _check(lib().adock_ligand_image(self.h, C.byref(n), C.byref(p), C.byref(m)))
        blob = bytes(np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_ubyte)), (n.value,)))
        return blob, np.ctypeslib.as_array(C.cast(m, C.POINTER(C.c_int)), (self.N,)).copy()

    def lane_image(self):
        """(host copy of the lane-per-individual image as bytes, pos_of_ext [N])"""
        n, p, m = C.c_int(), C.c_void_p(), C.c_void_p()
        _check(lib().adock_ligand_lane_image(self.h, C.byref(n), C.byref(p), C.byref(m)))
        blob = bytes(np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_ubyte)), (n.value,)))
        return blob, np.ctypeslib.as_array(C.cast(m, C.POINTER(C.c_int)), (self.N,)).copy()

    def close(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.adock_free_ligand(self.h)
            self.h = None

    __del__ = close


def adock_score_batch(grids: Grids, lig: Ligand, params, d_genotypes, d_energies, d_energy_terms=None, d_gradients=None):
    n, gs = d_genotypes.shape
    ds = d_gradients.shape[1] if d_gradients is not None else 0
    _check(lib().adock_score_batch(grids.h, lig.h, C.byref(params) if params is not None else None, _dp(d_genotypes), n, gs,
                                   _dp(d_energies), _dp(d_energy_terms), _dp(d_gradients), ds, _stream()))


def adock_score_batch_host(grids: Grids, lig: Ligand, params, h_genotypes, want_terms=True, want_grad=True):
    g = _np(h_genotypes, np.float32)
    n, gs = g.shape
    E = np.empty(n, np.float32)
    terms = np.empty((n, 2), np.float32) if want_terms else None
    grad = np.empty((n, 6 + lig.R), np.float32) if want_grad else None
    _check(lib().adock_score_batch_host(grids.h, lig.h, C.byref(params) if params is not None else None, _hp(g), n, gs, _hp(E),
                                        _hp(terms), _hp(grad), 6 + lig.R, None))
    return dict(E=E, terms=terms, grad=grad)


def adock_local_search(grids: Grids, lig: Ligand, params, d_genotypes, d_energies, d_iters=None, d_trace=None):
    n, gs = d_genotypes.shape
    if d_trace is not None:
        assert tuple(d_trace.shape) == (n, params.lsit)
    _check(lib().adock_local_search(grids.h, lig.h, C.byref(params) if params is not None else None, _dp(d_genotypes), n, gs,
                                    _dp(d_energies), _dp(d_iters), _dp(d_trace), _stream()))


def adock_local_search_noalloc(grids: Grids, lig: Ligand, params, d_genotypes, d_energies, d_iters=None, d_trace=None):
    """adock_local_search with the chain state in the library's static device array: no device allocation (adock.h)"""
    n, gs = d_genotypes.shape
    if d_trace is not None:
        assert tuple(d_trace.shape) == (n, params.lsit)
    _check(lib().adock_local_search_noalloc(grids.h, lig.h, C.byref(params) if params is not None else None, _dp(d_genotypes), n, gs,
                                            _dp(d_energies), _dp(d_iters), _dp(d_trace), _stream()))


def adock_solis_wets(grids: Grids, lig: Ligand, params, d_genotypes, d_energies, seed, generation, d_evals=None, d_trace=None):
    """d_energies: in (energies of the starting genotypes) / out (accepted energies)"""
    n, gs = d_genotypes.shape
    if d_trace is not None:
        assert tuple(d_trace.shape) == (n, params.lsit)
    _check(lib().adock_solis_wets(grids.h, lig.h, C.byref(params) if params is not None else None, _dp(d_genotypes), n, gs,
                                  _dp(d_energies), _dp(d_evals), _dp(d_trace), int(seed), int(generation), _stream()))


def adock_philox(key, d_ctr, d_out):
    k = _np(key, np.uint32)
    _check(lib().adock_philox(_hp(k), _dp(d_ctr), int(d_ctr.shape[0]), _dp(d_out), _stream()))


def adock_ga_generation(grids: Grids, lig: Ligand, params, nrun, P, generation, seed, d_pop, d_energies, d_newpop,
                        d_decisions=None, d_ls_picks=None) -> int:
    n_ls = C.c_int()
    _check(lib().adock_ga_generation(grids.h, lig.h, C.byref(params) if params is not None else None, int(nrun), int(P),
                                     int(generation), int(seed), _dp(d_pop), _dp(d_energies), _dp(d_newpop), _dp(d_decisions),
                                     _dp(d_ls_picks), C.byref(n_ls), _stream()))
    return n_ls.value


def adock_dock(grids: Grids, lig: Ligand, params, nrun, pop_size, max_evals, seed, want_coords=True):
    G = 7 + lig.R
    bg = np.zeros((nrun, G), np.float32)
    bE = np.zeros(nrun, np.float32)
    bx = np.zeros((nrun, lig.N, 3), np.float32) if want_coords else None
    ev = np.zeros(nrun, np.int64)
    gens = np.zeros(nrun, np.int32)
    _check(lib().adock_dock(grids.h, lig.h, C.byref(params) if params is not None else None, int(nrun), int(pop_size),
                            int(max_evals), int(seed), _hp(bg), _hp(bE), _hp(bx), _hp(ev), _hp(gens), _stream()))
    return dict(genotypes=bg, energies=bE, coords=bx, evals=ev, gens=gens)


def adock_dock_many(grids: Grids, ligs, params, nrun, pop_size, max_evals, seeds, want_coords=False):
    nlig = len(ligs)
    gs = max(7 + l.R for l in ligs)
    cs = max(l.N for l in ligs)
    handles = (C.c_void_p * nlig)(*[l.h for l in ligs])
    sd = _np(seeds, np.uint64)
    bg = np.zeros((nlig, nrun, gs), np.float32)
    bE = np.zeros((nlig, nrun), np.float32)
    bx = np.zeros((nlig, nrun, cs, 3), np.float32) if want_coords else None
    ev = np.zeros((nlig, nrun), np.int64)
    gens = np.zeros((nlig, nrun), np.int32)
    _check(lib().adock_dock_many(grids.h, C.cast(handles, C.c_void_p), nlig, C.byref(params) if params is not None else None,
                                 int(nrun), int(pop_size), int(max_evals), _hp(sd), gs, _hp(bg), _hp(bE), cs, _hp(bx), _hp(ev),
                                 _hp(gens), _stream()))
    return dict(genotypes=bg, energies=bE, coords=bx, evals=ev, gens=gens)


def adock_screen(grids: Grids, ligs, params, nrun, pop_size, max_evals, seeds, batch, host_threads=4):
    """ligs: workloads.Ligand objects sharing one force-field table (T, pair_coeffs, solpar, vol).  Host buffers in,
    host results out; returns dict(genotypes [nlig][nrun][G], energies, evals, stats)."""
    nlig = len(ligs)
    keep = []                                   # the arrays the descriptors point into
    desc = (adock_ligand_desc * max(nlig, 1))()
    for i, l in enumerate(ligs):
        a = [_np(l.xyz, np.float32), _np(l.type, np.int32), _np(l.charge, np.float32), _np(l.bonds, np.int32).reshape(-1, 2),
             _np(l.rot_bonds, np.int32).reshape(-1, 2)]
        keep.append(a)
        desc[i] = adock_ligand_desc(a[0].shape[0], _hp(a[0]), _hp(a[1]), _hp(a[2]), a[3].shape[0], _hp(a[3]), a[4].shape[0], _hp(a[4]),
                                    int(l.root_atom))
    l0 = ligs[0]
    co, sp, vo = _np(l0.pair_coeffs, np.float32), _np(l0.solpar, np.float32), _np(l0.vol, np.float32)
    gs = max(7 + a[4].shape[0] for a in keep)
    sd = _np(seeds, np.uint64)
    bg = np.zeros((nlig, nrun, gs), np.float32)
    bE = np.zeros((nlig, nrun), np.float32)
    ev = np.zeros((nlig, nrun), np.int64)
    st = adock_screen_stats()
    L = lib()
    L.adock_screen.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int,
                               C.c_longlong, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    _check(L.adock_screen(grids.h, C.addressof(params) if params is not None else None, int(l0.T), _hp(co), _hp(sp), _hp(vo), nlig,
                          C.addressof(desc), int(nrun), int(pop_size), int(max_evals), _hp(sd), int(batch), int(host_threads), gs,
                          _hp(bg), _hp(bE), _hp(ev), C.addressof(st), _stream()))
    return dict(genotypes=bg, energies=bE, evals=ev,
                stats={k: getattr(st, k) for k, _ in adock_screen_stats._fields_})


def adock_pose_rmsd(coords, ref=None, energies=None, tol=2.0, want_pairs=True):
    """coords host [n][N][3]; returns dict(rmsd_ref [n] or None, rmsd_pair [n][n] or None, cluster [n] or None, nclusters)"""
    x = _np(coords, np.float32)
    n, N = x.shape[0], x.shape[1]
    r = _np(ref, np.float32) if ref is not None else None
    E = _np(energies, np.float32) if energies is not None else None
    rr = np.zeros(n, np.float32) if r is not None else None
    rp = np.zeros((n, n), np.float32) if want_pairs else None
    cl = np.zeros(n, np.int32) if E is not None else None
    nc = C.c_int()
    L = lib()
    L.adock_pose_rmsd.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p,
                                  C.c_void_p, C.c_void_p]
    _check(L.adock_pose_rmsd(n, N, _hp(x), _hp(r), _hp(rr), _hp(rp), _hp(E), float(tol), _hp(cl), C.addressof(nc), _stream()))
    return dict(rmsd_ref=rr, rmsd_pair=rp, cluster=cl, nclusters=nc.value)


def adock_profile(enable: bool) -> None:
    _check(lib().adock_profile(1 if enable else 0))


def adock_profile_read() -> dict:
    ms, n, ev = C.c_double(), C.c_longlong(), C.c_longlong()
    _check(lib().adock_profile_read(C.byref(ms), C.byref(n), C.byref(ev)))
    return dict(ls_ms=ms.value, ls_launches=n.value, ls_evals=ev.value)


PATHS = {"auto": 0, "warp": 1, "lane": 2, "lane1": 21, "lane2": 22, "lane4": 24, "tm8": 41, "tm12": 42, "tm16": 43, "team": 3}


def adock_set_path(path) -> None:
    """kernel family: 'auto' (by problem size), 'warp' (warp per individual), 'lane' (lane per individual, warps per
    group of 32 individuals chosen by size), 'lane1' / 'lane2' / 'lane4' (that number of warps per group), 'tm8' / 'tm12' /
    'tm16' (one warp per group, atom positions in tensor memory, at most that many warps per SM) or 'team' (the
    ADADELTA chains of the dockings and of adock_local_search each run on a CTA of 4 warps; everything else as 'warp')"""
    _check(lib().adock_set_path(PATHS[path] if isinstance(path, str) else int(path)))


def adock_last_dock_path() -> str:
    return {0: "none", 1: "warp", 2: "lane", 3: "team"}[int(lib().adock_last_dock_path())]


def adock_alu_peak() -> dict:
    """measured FP32 peak of this device (include/adock.h): dict(tflops, fma_lanes_per_clk_sm)"""
    t, l = C.c_double(), C.c_double()
    lib().adock_alu_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p]
    _check(lib().adock_alu_peak(C.byref(t), C.byref(l), _stream()))
    return dict(tflops=t.value, fma_lanes_per_clk_sm=l.value)


def adock_tmem_probe(warps: int, mode: int, iters: int = 20000) -> dict:
    """tensor memory as per-lane scratch (include/adock.h): dict(errors, cycles_per_iteration)"""
    err, cyc = C.c_int(), C.c_double()
    lib().adock_tmem_probe.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double), C.c_void_p]
    _check(lib().adock_tmem_probe(int(warps), int(mode), int(iters), C.byref(err), C.byref(cyc), _stream()))
    return dict(errors=err.value, cycles_per_iteration=cyc.value)


def adock_launch_count(reset: bool = False) -> int:
    return int(lib().adock_launch_count(1 if reset else 0))
