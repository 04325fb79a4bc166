"""ctypes wrapper of the CPU oracle (oracle/adock_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It shares nothing with paper_2007_03678_b200 (the CUDA path) and never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "adock_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_LIB32 = os.path.join(_HERE, "liboracle_f32.so")
_lib = None
_lib32 = None


def build(force: bool = False) -> str:
    """liboracle.so = the oracle (fp64).  liboracle_f32.so = the same source with the score path (R3-R6) in honest
    fp32 (-DORC_REAL=float): a measuring stick for tolerances, never a parity reference."""
    for out, extra in ((_LIB, []), (_LIB32, ["-DORC_REAL=float"])):
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
                                   *extra, "-o", out, _SRC])
    return _LIB


class OPar(C.Structure):
    _fields_ = [(k, C.c_double) for k in (
        "elec_scale", "diel_A", "diel_B", "diel_k", "diel_lambda", "w_desolv", "ds_sigma", "qasp", "r_min", "k_wall",
        "ad_rho", "ad_eps", "lsrat", "tourn_prob", "xover_rate", "mut_rate", "dmov", "dang",
        "sw_rho0", "sw_rho_lb", "sw_expand", "sw_contract", "sw_bias_keep", "sw_bias_gain", "sw_bias_decay", "as_tol")] + [
        (k, C.c_int) for k in ("lsit", "max_gens", "ls_method", "sw_max_succ", "sw_max_fail", "autostop", "as_window")]


# GA probabilities and step sizes are float32 parameters of the method: both sides see the same
# float32 value (decisions u < p are then identical), so round them once here.
_F32_FIELDS = ("lsrat", "tourn_prob", "xover_rate", "mut_rate", "dmov", "dang",
               "sw_rho0", "sw_rho_lb", "sw_expand", "sw_contract", "sw_bias_keep", "sw_bias_gain", "sw_bias_decay", "as_tol")


def params(d: dict) -> OPar:
    p = OPar()
    for k, _ in OPar._fields_:
        v = d[k]
        if k in _F32_FIELDS:
            v = float(np.float32(v))
        setattr(p, k, v)
    return p


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_dock.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(OPar), C.c_int, C.c_int, C.c_longlong, C.c_ulonglong,
                                  C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
    return _lib


def lib_f32():
    """the fp32 build of the score path; handles (Ligand, Grids) of the fp64 library are valid in it (same structs)"""
    global _lib32
    if _lib32 is None:
        build()
        _lib32 = C.CDLL(_LIB32)
        assert _lib32.orc_real_bytes() == 4 and lib().orc_real_bytes() == 8
    return _lib32


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, np.float32)


def _i32(a):
    return np.ascontiguousarray(a, np.int32)


def _f64(a):
    return np.ascontiguousarray(a, np.float64)


class Ligand:
    def __init__(self, xyz, type, charge, bonds, rot_bonds, root_atom, T, pair_coeffs, solpar, vol):
        xyz, type, charge = _f32(xyz), _i32(type), _f32(charge)
        bonds, rot = _i32(bonds).reshape(-1, 2), _i32(rot_bonds).reshape(-1, 2)
        self.N, self.R, self.T = xyz.shape[0], rot.shape[0], int(T)
        self._h = C.c_void_p()
        rc = lib().orc_lig_create(self.N, _p(xyz), _p(type), _p(charge), bonds.shape[0], _p(bonds), self.R, _p(rot),
                                  int(root_atom), self.T, _p(_f32(pair_coeffs)), _p(_f32(solpar)), _p(_f32(vol)),
                                  C.byref(self._h))
        if rc != 0:
            raise ValueError("oracle: invalid ligand")
        npairs, nfrag = C.c_int(), C.c_int()
        lib().orc_lig_info(self._h, C.byref(npairs), C.byref(nfrag))
        self.npairs, self.nfrag = npairs.value, nfrag.value
        self.pairs = np.zeros((self.npairs, 2), np.int32)
        self.tor_order = np.zeros(self.R, np.int32)
        self.moved = np.zeros((self.R, self.N), np.uint8)
        self.depth = np.zeros(self.R, np.int32)
        self.frag = np.zeros(self.N, np.int32)
        self.rot = np.zeros((self.R, 2), np.int32)
        self.pivot = np.zeros(3, np.float64)
        self.dist = np.zeros((self.N, self.N), np.int32)
        lib().orc_lig_get(self._h, _p(self.pairs), _p(self.tor_order), _p(self.moved), _p(self.depth), _p(self.frag),
                          _p(self.rot), _p(self.pivot), _p(self.dist))

    @classmethod
    def from_workload(cls, lig):
        return cls(lig.xyz, lig.type, lig.charge, lig.bonds, lig.rot_bonds, lig.root_atom, lig.T, lig.pair_coeffs,
                   lig.solpar, lig.vol)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_lig_free(self._h)
            self._h = None

    def identity_genotype(self):
        g = np.zeros(7 + self.R, np.float64)
        g[0:3] = self.pivot
        g[3] = 1.0
        return g

    def pose(self, geno):
        geno = _f64(geno)
        assert geno.shape == (7 + self.R,)
        out = np.zeros((self.N, 3), np.float64)
        if lib().orc_pose(self._h, _p(geno), _p(out)) != 0:
            raise ValueError("oracle: degenerate quaternion")
        return out


class Grids:
    def __init__(self, maps, spacing, origin):
        maps = _f32(maps)
        self.M, self.nz, self.ny, self.nx = maps.shape
        self.spacing = float(spacing)
        self.origin = _f32(origin)
        self._h = C.c_void_p()
        rc = lib().orc_grid_create(_p(maps), self.M, self.nx, self.ny, self.nz, C.c_double(self.spacing), _p(self.origin),
                                   C.byref(self._h))
        if rc != 0:
            raise ValueError("oracle: invalid grids")

    @classmethod
    def from_workload(cls, g):
        return cls(g.maps, g.spacing, g.origin)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_grid_free(self._h)
            self._h = None

    def trilinear(self, m, xyz, grad=True):
        xyz = _f64(xyz).reshape(-1, 3)
        val = np.zeros(xyz.shape[0], np.float64)
        g = np.zeros((xyz.shape[0], 3), np.float64) if grad else None
        if lib().orc_trilinear(self._h, int(m), _p(xyz), xyz.shape[0], _p(val), _p(g)) != 0:
            raise ValueError("bad map index")
        return (val, g) if grad else val

    def grid_atom(self, par: OPar, type_, q, T, x):
        x = _f64(x)
        E = C.c_double()
        g = np.zeros(3, np.float64)
        lib().orc_grid_atom(self._h, C.byref(par), int(type_), C.c_double(q), int(T), _p(x), C.byref(E), _p(g))
        return E.value, g


def pair_energy(par: OPar, c12, cA, expA, qq, dsco, d):
    E, dE = C.c_double(), C.c_double()
    lib().orc_pair_energy(C.byref(par), C.c_double(c12), C.c_double(cA), C.c_double(expA), C.c_double(qq), C.c_double(dsco),
                          C.c_double(d), C.byref(E), C.byref(dE))
    return E.value, dE.value


def score(grids: Grids, lig: Ligand, par: OPar, genos, want_grad=True, nthreads=0, fp32=False):
    """float32 genotypes [n, >=7+R] -> dict(E[n], terms[n,2], grad[n,6+R], margins[n,2], scales[n,3]) in float64.
    fp32=True runs the same statements in float (liboracle_f32.so): how far honest fp32 lands from the oracle."""
    genos = _f32(genos)
    if genos.ndim == 1:
        genos = genos[None]
    n, gs = genos.shape
    E = np.zeros(n, np.float64)
    terms = np.zeros((n, 2), np.float64)
    grad = np.zeros((n, 6 + lig.R), np.float64) if want_grad else None
    margins = np.zeros((n, 2), np.float64)
    scales = np.zeros((n, 3), np.float64)
    rc = (lib_f32() if fp32 else lib()).orc_score(grids._h, lig._h, C.byref(par), _p(genos), n, gs, _p(E), _p(terms), _p(grad),
                                                  _p(margins), _p(scales), int(nthreads))
    if rc != 0:
        raise ValueError("oracle: ligand types exceed grid maps")
    return dict(E=E, terms=terms, grad=grad, margins=margins, scales=scales)


def score_f64(grids: Grids, lig: Ligand, par: OPar, geno, want_grad=True):
    """one float64 genotype -> (E, grad) with no float32 rounding of the input (finite-difference pins)."""
    geno = _f64(geno)
    E = C.c_double()
    grad = np.zeros(6 + lig.R, np.float64) if want_grad else None
    lib().orc_score_f64(grids._h, lig._h, C.byref(par), _p(geno), C.byref(E), _p(grad))
    return E.value, grad


_FN = C.CFUNCTYPE(C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)


def adadelta_rn(x0, fn, rho, eps, iters):
    """generic R^n ADADELTA; fn(x)->(f, grad). Returns (x_final, trace of f before each step)."""
    x = _f64(x0).copy()
    n = x.shape[0]

    def cb(n_, xp, gp, _user):
        xv = np.ctypeslib.as_array(xp, (n_,))
        f, g = fn(xv.copy())
        np.ctypeslib.as_array(gp, (n_,))[:] = g
        return float(f)

    trace = np.zeros(iters, np.float64)
    lib().orc_adadelta_rn(n, _p(x), C.c_double(rho), C.c_double(eps), int(iters), _FN(cb), None, _p(trace))
    return x, trace


def apply_step(R, x, delta):
    x = _f64(x).copy()
    lib().orc_apply_step(int(R), _p(x), _p(_f64(delta)))
    return x


def adadelta(grids: Grids, lig: Ligand, par: OPar, geno, trace=False, fp32=False):
    """docking local search from one genotype: (best genotype, best E, iterations used[, traceE, traceX]).
    fp32=True: the same statements with the score path in float (liboracle_f32.so): how fast an honest fp32 chain parts
    from the oracle's (a measuring stick for the trace tolerance, never a parity reference)."""
    g = _f64(geno).copy()
    E = C.c_double(float("nan"))
    it = C.c_int()
    tE = np.full(par.lsit, np.nan) if trace else None
    tX = np.full((par.lsit, 7 + lig.R), np.nan) if trace else None
    (lib_f32() if fp32 else lib()).orc_adadelta(grids._h, lig._h, C.byref(par), _p(g), C.byref(E), C.byref(it), _p(tE), _p(tX))
    return (g, E.value, it.value, tE, tX) if trace else (g, E.value, it.value)


def solis_wets_rn(x0, E0, fn, amp, par: OPar, seed, id, gen):
    """generic R^n Solis-Wets (R11); fn(x)->f. Returns (x, E, evals, iterations, final rho, trace of E after each iteration)."""
    x = _f64(x0).copy()
    n = x.shape[0]

    def cb(n_, xp, _gp, _user):
        return float(fn(np.ctypeslib.as_array(xp, (n_,)).copy()))

    E = C.c_double(float(E0)); it = C.c_int(); rho = C.c_double()
    tE = np.full(par.lsit, np.nan)
    L = lib()
    L.orc_solis_wets_rn.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_ulonglong, C.c_uint, C.c_uint,
                                    _FN, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    ev = L.orc_solis_wets_rn(n, _p(x), C.addressof(E), _p(_f64(amp)), C.addressof(par), int(seed), int(id), int(gen), _FN(cb), None,
                             C.addressof(it), C.addressof(rho), _p(tE))
    return x, E.value, ev, it.value, rho.value, tE


def solis_wets(grids: Grids, lig: Ligand, par: OPar, geno, E0, seed, id, gen):
    """docking Solis-Wets from one genotype with carried energy E0: (genotype, E, evals, iterations, rho, traceE)."""
    g = _f64(geno).copy()
    E = C.c_double(float(E0)); it = C.c_int(); rho = C.c_double()
    tE = np.full(par.lsit, np.nan)
    L = lib()
    L.orc_solis_wets.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_ulonglong, C.c_uint, C.c_uint, C.c_void_p, C.c_void_p,
                                 C.c_void_p, C.c_void_p, C.c_void_p]
    ev = L.orc_solis_wets(grids._h, lig._h, C.addressof(par), int(seed), int(id), int(gen), _p(g), C.addressof(E),
                          C.addressof(it), C.addressof(rho), _p(tE))
    return g, E.value, ev, it.value, rho.value, tE


def philox(key, ctr):
    key = np.ascontiguousarray(key, np.uint32)
    ctr = np.ascontiguousarray(ctr, np.uint32).reshape(-1, 4)
    out = np.zeros_like(ctr)
    lib().orc_philox(_p(key), _p(ctr), ctr.shape[0], _p(out))
    return out


def ga_init(grids: Grids, R, seed, run, P):
    pop = np.zeros((P, 7 + R), np.float64)
    lib().orc_ga_init(grids._h, int(R), C.c_ulonglong(seed), int(run), int(P), _p(pop))
    return pop


def ga_offspring(par: OPar, R, run, gen, seed, pop, E):
    pop, E = _f64(pop), _f64(E)
    P = pop.shape[0]
    newpop = np.zeros_like(pop)
    newE = np.zeros(P, np.float64)
    dec = np.zeros((P, 10), np.int32)
    lib().orc_ga_offspring(C.byref(par), P, int(R), int(run), int(gen), C.c_ulonglong(seed), _p(pop), _p(E), _p(newpop),
                           _p(newE), _p(dec))
    return newpop, newE, dec


def ls_pick(par: OPar, P, run, gen, seed):
    picks = np.zeros(P, np.int32)
    n = lib().orc_ls_pick(C.byref(par), int(P), int(run), int(gen), C.c_ulonglong(seed), _p(picks))
    return picks[:n].copy()


def dock(grids: Grids, lig: Ligand, par: OPar, nrun, pop_size, max_evals, seed, hist_len=0, nthreads=0):
    G = 7 + lig.R
    bg = np.zeros((nrun, G), np.float64)
    bE = np.zeros(nrun, np.float64)
    bx = np.zeros((nrun, lig.N, 3), np.float64)
    ev = np.zeros(nrun, np.int64)
    gens = np.zeros(nrun, np.int32)
    hist = np.zeros((nrun, hist_len), np.float64) if hist_len else None
    rc = lib().orc_dock(grids._h, lig._h, C.byref(par), int(nrun), int(pop_size), int(max_evals), int(seed), _p(bg), _p(bE),
                        _p(bx), _p(ev), _p(gens), _p(hist), int(hist_len), int(nthreads))
    if rc != 0:
        raise ValueError("oracle: invalid dock arguments")
    return dict(genotypes=bg, energies=bE, coords=bx, evals=ev, gens=gens, history=hist)


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ------------------------------------------------------------------ R13 pose post-processing (RMSD)
def pose_rmsd(a, b):
    """sqrt(mean_i |a_i - b_i|^2): same atom order, no superposition, no symmetry correction.  a [..., N, 3], b [N, 3]"""
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return np.sqrt(((a - b) ** 2).sum(-1).mean(-1))


def pose_rmsd_pairs(x):
    x = np.asarray(x, np.float64)
    return np.array([[pose_rmsd(x[i], x[j]) for j in range(x.shape[0])] for i in range(x.shape[0])])


def cluster_poses(energies, pair, tol):
    """poses in order of increasing energy (ties: lower index); a pose joins the first cluster (creation order) whose seed
    is within tol, else it seeds a new one [LIT: AutoDock's RMSD-tolerance clustering].  Returns (cluster id per pose, n)."""
    order = sorted(range(len(energies)), key=lambda k: (energies[k], k))
    seeds, out = [], [0] * len(energies)
    for k in order:
        for c, s in enumerate(seeds):
            if pair[k][s] <= tol:
                out[k] = c
                break
        else:
            out[k] = len(seeds)
            seeds.append(k)
    return np.array(out, np.int32), len(seeds)
