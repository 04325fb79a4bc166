"""Seeded synthetic inputs (ligands, grid maps, genotypes) shaped like the paper's workloads.

This module is the ONLY code that serves both the CPU oracle (oracle/) and the CUDA path: it
produces plain numpy arrays that are handed unchanged to both.  It implements none of the
method's arithmetic (no pose building, no interpolation, no pair sums, no GA/ADADELTA); what it
does compute are the *inputs*: pseudo-receptor fields sampled on a lattice, and force-field
tables.  Recipe: DESIGN.md "Input recipe" (BASELINE.json configs).

The paper's own datasets (S42, SN9000, Mpro) are not available;
these inputs stand in for them (box sizes follow PAPER.md lines 116, 148-150, 225).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# AutoDock4 free-energy weights (literature values; exposed as parameters, see DESIGN.md readings)
W_VDW, W_HB, W_EL, W_DS = 0.1662, 0.1209, 0.1406, 0.1322
ELEC_K = 332.06363
DIEL_A, DIEL_B, DIEL_K, DIEL_LAMBDA = -8.5525, 86.9525, 7.7839, 0.003627
DS_SIGMA = 3.6

# every tunable constant of the method, by name; each side packs it into its own struct
DEFAULT_PARAMS = dict(
    elec_scale=W_EL * ELEC_K, diel_A=DIEL_A, diel_B=DIEL_B, diel_k=DIEL_K, diel_lambda=DIEL_LAMBDA,
    w_desolv=W_DS, ds_sigma=DS_SIGMA, qasp=0.01097, r_min=0.5, k_wall=1000.0,
    ad_rho=0.8, ad_eps=1e-2, lsit=300, lsrat=0.06,
    tourn_prob=0.60, xover_rate=0.80, mut_rate=0.02, dmov=2.0, dang=math.pi / 2, max_gens=27000,
    # R11 Solis-Wets [LIT] and R12 autostop [CHOICE]; ls_method 0 = ADADELTA, 1 = Solis-Wets
    ls_method=0, sw_rho0=1.0, sw_rho_lb=0.01, sw_expand=2.0, sw_contract=0.5, sw_bias_keep=0.6, sw_bias_gain=0.4,
    sw_bias_decay=0.5, sw_max_succ=4, sw_max_fail=4, autostop=0, as_window=10, as_tol=0.15,
)


@dataclass
class Ligand:
    xyz: np.ndarray          # [N,3] float32, grid frame (Angstrom)
    type: np.ndarray         # [N] int32 in [0,T)
    charge: np.ndarray       # [N] float32
    bonds: np.ndarray        # [nbonds,2] int32
    rot_bonds: np.ndarray    # [R,2] int32
    root_atom: int
    T: int
    pair_coeffs: np.ndarray  # [T,T,4] float32: c12, cA, expA (6 or 10), 0
    solpar: np.ndarray       # [T] float32
    vol: np.ndarray          # [T] float32

    @property
    def N(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def R(self) -> int:
        return int(self.rot_bonds.shape[0])


@dataclass
class GridSet:
    maps: np.ndarray         # [M,nz,ny,nx] float32, M = T+2 (types, elec, desolv)
    spacing: float
    origin: np.ndarray       # [3] float32 (x,y,z of node (0,0,0))
    meta: dict = field(default_factory=dict)

    @property
    def M(self) -> int:
        return int(self.maps.shape[0])

    @property
    def dims(self):
        return int(self.maps.shape[3]), int(self.maps.shape[2]), int(self.maps.shape[1])  # nx,ny,nz

    @property
    def box_lo(self) -> np.ndarray:
        return self.origin.astype(np.float64)

    @property
    def box_hi(self) -> np.ndarray:
        nx, ny, nz = self.dims
        return self.origin.astype(np.float64) + self.spacing * np.array([nx - 1, ny - 1, nz - 1], np.float64)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def make_type_params(T: int, seed: int):
    """Per-type LJ radius/well depth, volume, solvation parameter -> weighted pair table."""
    g = _rng(1000003 * seed + 17)
    Rii = g.uniform(3.0, 4.5, T)
    eii = g.uniform(0.02, 0.30, T)
    solpar = g.uniform(-0.003, 0.001, T)
    vol = (4.0 / 3.0) * math.pi * (Rii / 2.0) ** 3
    coeffs = np.zeros((T, T, 4), np.float64)
    for a in range(T):
        for b in range(T):
            Rab = 0.5 * (Rii[a] + Rii[b])
            eab = math.sqrt(eii[a] * eii[b])
            hb = T >= 2 and {a, b} == {T - 1, T - 2}
            if hb:      # one 12-10 hydrogen-bond type pair
                Rab, eab = 1.9, 5.0
                coeffs[a, b] = (W_HB * 5.0 * eab * Rab ** 12, W_HB * 6.0 * eab * Rab ** 10, 10.0, 0.0)
            else:
                coeffs[a, b] = (W_VDW * eab * Rab ** 12, W_VDW * 2.0 * eab * Rab ** 6, 6.0, 0.0)
    return Rii, eii, coeffs.astype(np.float32), solpar.astype(np.float32), vol.astype(np.float32)


def make_ligand(N: int, R: int, T: int, seed: int, centre=(0.0, 0.0, 0.0), far_sep: float | None = None,
                max_deg: int = 4) -> Ligand:
    """Random bonded tree, 1.5 A bonds, degree <= max_deg, atoms >= 1.3 A apart; R rotatable bonds drawn
    from bonds whose two ends both have degree >= 2 (all of them if fewer than R exist).
    far_sep (the non-clashing variant): atoms four or more bonds apart are also kept at least
    far_sep Angstrom apart in the input conformation, so that no non-excluded pair starts inside its repulsive wall."""
    g = _rng(seed)
    xyz = np.zeros((N, 3), np.float64)
    deg = np.zeros(N, np.int64)
    topo = np.zeros((N, N), np.int64)                   # bond-count distance in the tree built so far
    bonds = []
    for k in range(1, N):
        best, best_pos, best_p = -np.inf, None, None
        for _ in range(200 if far_sep is None else 2000):
            cand = np.flatnonzero(deg[:k] < max_deg)
            p = int(cand[g.integers(len(cand))])
            d = g.normal(size=3)
            d /= np.linalg.norm(d)
            pos = xyz[p] + 1.5 * d
            dist = np.linalg.norm(xyz[:k] - pos, axis=1)
            dist[p] = np.inf
            if far_sep is None:
                if dist.min() >= 1.3:
                    break
                continue
            far = topo[p, :k] + 1 >= 4
            slack = min(dist.min() - 1.3, (dist[far].min() - far_sep) if far.any() else np.inf)
            if slack > best:
                best, best_pos, best_p = slack, pos, p
            if slack >= 0:
                break
        if far_sep is not None:
            pos, p = best_pos, best_p
        xyz[k] = pos
        topo[k, :k] = topo[p, :k] + 1
        topo[:k, k] = topo[k, :k]
        deg[p] += 1
        deg[k] += 1
        bonds.append((p, k))
    bonds = np.array(bonds, np.int32).reshape(-1, 2)
    eligible = [b for b in range(len(bonds)) if deg[bonds[b, 0]] >= 2 and deg[bonds[b, 1]] >= 2]
    pick = g.permutation(len(eligible))[: min(R, len(eligible))]
    rot = bonds[np.sort(np.array([eligible[i] for i in pick], np.int64))].reshape(-1, 2)
    types = g.integers(0, T, N).astype(np.int32)
    charge = np.clip(g.normal(0.0, 0.2, N), -1.0, 1.0).astype(np.float32)
    xyz = xyz - xyz.mean(axis=0) + np.asarray(centre, np.float64)
    _, _, coeffs, solpar, vol = make_type_params(T, seed)
    return Ligand(xyz.astype(np.float32), types, charge, bonds, rot.astype(np.int32), 0, T, coeffs, solpar, vol)


def make_chain_ligand(N: int, T: int = 2, seed: int = 0, centre=(0.0, 0.0, 0.0)) -> Ligand:
    """Zig-zag linear chain 0-1-...-(N-1); every interior bond (k,k+1), 1<=k<=N-3, rotatable.
    Hand-countable topology used by the preprocessing pins."""
    xyz = np.zeros((N, 3), np.float64)
    for k in range(1, N):
        xyz[k] = xyz[k - 1] + 1.5 * np.array([math.cos(0.6 * (-1) ** k), math.sin(0.6 * (-1) ** k), 0.15 * (k % 3)])
    bonds = np.array([(k, k + 1) for k in range(N - 1)], np.int32)
    rot = np.array([(k, k + 1) for k in range(1, N - 2)], np.int32).reshape(-1, 2)
    g = _rng(seed + 99)
    types = g.integers(0, T, N).astype(np.int32)
    charge = np.clip(g.normal(0.0, 0.2, N), -1.0, 1.0).astype(np.float32)
    xyz = xyz - xyz.mean(axis=0) + np.asarray(centre, np.float64)
    _, _, coeffs, solpar, vol = make_type_params(T, seed)
    return Ligand(xyz.astype(np.float32), types, charge, bonds, rot, 0, T, coeffs, solpar, vol)


def make_grids(n: int | tuple, T: int, K: int, pocket_radius: float, seed: int, spacing: float = 0.375,
               chunk: int = 16384) -> GridSet:
    """M = T+2 maps on an nx*ny*nz lattice from K random pseudo-receptor atoms (12-6 LJ per ligand
    type, screened Coulomb potential, Gaussian desolvation), r floored at 0.5 A, values clamped to
    +1e5 (BASELINE.json configs).  Evaluated in float64 (torch CPU, or CUDA when present), cast to fp32."""
    import torch

    nx, ny, nz = (n, n, n) if isinstance(n, int) else n
    g = _rng(7919 * seed + 5)
    edge = spacing * np.array([nx - 1, ny - 1, nz - 1], np.float64)
    origin = np.zeros(3, np.float64)
    centre = origin + 0.5 * edge
    pos = np.empty((0, 3))
    while len(pos) < K:
        c = g.uniform(0.0, 1.0, (2 * K + 16, 3)) * edge + origin
        c = c[np.linalg.norm(c - centre, axis=1) >= pocket_radius]
        pos = np.concatenate([pos, c])[:K]
    Rii, eii, _, _, _ = make_type_params(T, seed)       # ligand-side type parameters of this config
    gk = _rng(7919 * seed + 6)
    rt = gk.integers(0, T, K)
    rq = gk.normal(0.0, 0.3, K)
    rR, re_, rvol = Rii[rt], eii[rt], (4.0 / 3.0) * math.pi * (Rii[rt] / 2.0) ** 3
    # coefficient matrices [K, T]: field of type t = sum_K A[K,t] r^-12 - B[K,t] r^-6
    Rtk = 0.5 * (Rii[None, :] + rR[:, None])
    etk = np.sqrt(eii[None, :] * re_[:, None])
    A = W_VDW * etk * Rtk ** 12
    B = W_VDW * 2.0 * etk * Rtk ** 6

    dev = torch.device("cuda" if torch.cuda.is_available() else "cpu")
    f64 = torch.float64
    tpos = torch.tensor(pos, dtype=f64, device=dev)
    tA, tB = torch.tensor(A, dtype=f64, device=dev), torch.tensor(B, dtype=f64, device=dev)
    tq, tv = torch.tensor(rq, dtype=f64, device=dev), torch.tensor(rvol, dtype=f64, device=dev)
    iz, iy, ix = torch.meshgrid(torch.arange(nz, device=dev), torch.arange(ny, device=dev),
                                torch.arange(nx, device=dev), indexing="ij")
    pts = torch.stack([ix, iy, iz], -1).reshape(-1, 3).to(f64) * spacing + torch.tensor(origin, dtype=f64, device=dev)
    out = torch.empty((T + 2, pts.shape[0]), dtype=f64, device=dev)
    for s in range(0, pts.shape[0], chunk):
        p = pts[s:s + chunk]
        r = torch.cdist(p, tpos).clamp_min(0.5)                     # [chunk, K]
        r6 = r ** -6
        out[:T, s:s + chunk] = ((r6 * r6) @ tA - r6 @ tB).T
        eps_r = DIEL_A + DIEL_B / (1.0 + DIEL_K * torch.exp(-DIEL_LAMBDA * DIEL_B * r))
        out[T, s:s + chunk] = (W_EL * ELEC_K / (eps_r * r)) @ tq
        out[T + 1, s:s + chunk] = (W_DS * torch.exp(-r * r / (2 * DS_SIGMA ** 2))) @ tv
    maps = out.clamp_max(1e5).to(torch.float32).reshape(T + 2, nz, ny, nx).cpu().numpy()
    return GridSet(np.ascontiguousarray(maps), float(spacing), origin.astype(np.float32),
                   dict(K=K, pocket_radius=pocket_radius, seed=seed))


def make_affine_grids(n: int, T: int, coef, spacing: float = 0.375) -> GridSet:
    """Every map m is the affine field a_m*ix + b_m*iy + c_m*iz + d_m (coef: [T+2,4]); pin helper."""
    coef = np.asarray(coef, np.float64).reshape(T + 2, 4)
    iz, iy, ix = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    maps = np.stack([c[0] * ix + c[1] * iy + c[2] * iz + c[3] for c in coef]).astype(np.float32)
    return GridSet(np.ascontiguousarray(maps), float(spacing), np.zeros(3, np.float32), dict(affine=True))


def make_genotypes(n: int, R: int, grids: GridSet, seed: int, wall_tail: float = 0.01) -> np.ndarray:
    """[n, 7+R] float32: t uniform in the central 50% of the box, q = normalised N(0,1)^4,
    tau ~ U[-pi,pi); a wall_tail fraction has t within 1.5 A of (or beyond) a face."""
    g = _rng(31337 * seed + 3)
    lo, hi = grids.box_lo, grids.box_hi
    c, e = 0.5 * (lo + hi), hi - lo
    G = np.empty((n, 7 + R), np.float64)
    G[:, 0:3] = c + (g.uniform(-0.25, 0.25, (n, 3))) * e
    q = g.normal(size=(n, 4))
    G[:, 3:7] = q / np.linalg.norm(q, axis=1, keepdims=True)
    G[:, 7:] = g.uniform(-math.pi, math.pi, (n, R))
    ntail = int(round(wall_tail * n)) if n >= 100 else 0
    if ntail:
        rows = g.choice(n, ntail, replace=False)
        axis = g.integers(0, 3, ntail)
        side = g.integers(0, 2, ntail)
        off = g.uniform(-1.5, 1.5, ntail)
        G[rows, axis] = np.where(side == 0, lo[axis] + off, hi[axis] + off)
    return G.astype(np.float32)


def make_pocket_genotypes(n: int, R: int, grids: GridSet, seed: int, sigma_t: float = 1.0, sigma_tau: float = 0.25) -> np.ndarray:
    """[n, 7+R] float32 poses NEAR the input conformation inside the carved pocket: t = box centre + N(0, sigma_t) A,
    q uniform (normalised N(0,1)^4), tau ~ N(0, sigma_tau) rad.  With a far_sep ligand these are the non-clashing
    poses (energies O(1..100) kcal/mol, like a real complex) of DESIGN.md section 4."""
    g = _rng(271828 * seed + 11)
    c = 0.5 * (grids.box_lo + grids.box_hi)
    G = np.empty((n, 7 + R), np.float64)
    G[:, 0:3] = c + g.normal(0.0, sigma_t, (n, 3))
    q = g.normal(size=(n, 4))
    G[:, 3:7] = q / np.linalg.norm(q, axis=1, keepdims=True)
    G[:, 7:] = g.normal(0.0, sigma_tau, (n, R))
    return G.astype(np.float32)


# ---- the named configurations of BASELINE.json -------------------------------------------------
CONFIGS = {
    # name: ligand (N, R, T), grid n, receptor atoms K, pocket radius, seed
    "tiny":      dict(N=16, R=2, T=4, n=24, K=30, pocket=0.0, seed=0),
    "drug":      dict(N=40, R=8, T=7, n=64, K=2000, pocket=8.0, seed=1),
    "screen":    dict(N=None, R=None, T=7, n=80, K=4000, pocket=8.0, seed=2),
    "large":     dict(N=128, R=32, T=8, n=126, K=12000, pocket=8.0, seed=3),
    "sweep16":   dict(N=16, R=2, T=4, n=64, K=2000, pocket=8.0, seed=4),
    "sweep40":   dict(N=40, R=8, T=7, n=64, K=2000, pocket=8.0, seed=4),
    "sweep80":   dict(N=80, R=16, T=8, n=64, K=2000, pocket=8.0, seed=4),
    "sweep128":  dict(N=128, R=32, T=8, n=64, K=2000, pocket=8.0, seed=4),
}


def make_config(name: str, grid_n: int | None = None):
    """(GridSet, Ligand) of a named config; the ligand centroid sits at the box centre."""
    c = CONFIGS[name]
    n = grid_n or c["n"]
    grids = make_grids(n, c["T"], c["K"] if grid_n is None else max(30, int(c["K"] * (n / c["n"]) ** 3)),
                       min(c["pocket"], 0.3 * 0.375 * n), c["seed"])
    centre = 0.5 * (grids.box_lo + grids.box_hi)
    lig = make_ligand(c["N"], c["R"], c["T"], c["seed"], centre) if c["N"] else None
    return grids, lig


def make_screen_ligands(count: int, grids: GridSet, T: int = 7, seed: int = 2):
    """Virtual-screen ligand stream: atoms uniform in 15..60, rotatable bonds uniform in 0..15."""
    centre = 0.5 * (grids.box_lo + grids.box_hi)
    out = []
    for i in range(count):
        g = _rng(seed + i)
        out.append(make_ligand(int(g.integers(15, 61)), int(g.integers(0, 16)), T, seed + i, centre))
    return out


def share_type_table(ligs):
    """the same ligands with ONE force-field table (that of the first): a screen uses one atom-type table"""
    import dataclasses
    l0 = ligs[0]
    return [dataclasses.replace(l, pair_coeffs=l0.pair_coeffs, solpar=l0.solpar, vol=l0.vol) for l in ligs]


def shard(n_items: int, rank: int, world: int):
    """Ligand indices owned by `rank` (round-robin; the path shards with no exchange step)."""
    return list(range(rank, n_items, world))
