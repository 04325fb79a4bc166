"""Readers (and matching writers) for the two input file kinds the paper's program consumes (PAPER.md lines 100, 116:
"ligand files" in PDBQT form and the AutoGrid affinity / electrostatic / desolvation ".map" grids) -- SURVEY.md
section 8(f) NEXT-5.  Host-side input parsing only: they produce the arrays `adock_load_grids` / `adock_load_ligand` /
`adock_screen` take; none of the method's arithmetic lives here.  The container holds no real files, so the tests
round-trip synthetic ligands and maps through the writers below.

PDBQT ligand (public AutoDock format, fixed columns like PDB):
    ROOT / ENDROOT                      atoms of the root fragment
    BRANCH a b / ENDBRANCH a b          rotatable bond between atom serials a (nearer the root) and b; nested
    ATOM / HETATM records               serial 7-11, x 31-38, y 39-46, z 47-54, partial charge 67-76, atom type 78-79
    CONECT a b ...                      optional bonds (PDB standard); without them bonds are inferred from distances
    TORSDOF n
Grid map (public AutoGrid format): header lines GRID_PARAMETER_FILE, GRID_DATA_FILE, MACROMOLECULE, SPACING h,
NELEMENTS ex ey ez (numbers of INTERVALS: points = e+1 per axis), CENTER cx cy cz; then one value per line, x fastest,
then y, then z.
"""
from __future__ import annotations

import numpy as np

from .workloads import GridSet, Ligand

# single-bond covalent radii (Angstrom) by element, used only when a PDBQT file carries no CONECT records
_COVALENT = {"H": 0.31, "C": 0.76, "N": 0.71, "O": 0.66, "F": 0.57, "P": 1.07, "S": 1.05, "CL": 1.02, "BR": 1.20, "I": 1.39}
# AutoDock atom-type names -> element (aromatic carbon A, acceptor types NA / OA / SA, donor hydrogen HD ...)
_ELEMENT = {"A": "C", "NA": "N", "NS": "N", "OA": "O", "OS": "O", "SA": "S", "HD": "H", "HS": "H", "CL": "CL", "BR": "BR"}


def _element(atype: str) -> str:
    t = atype.upper()
    return _ELEMENT.get(t, t if t in _COVALENT else t[:1])


def read_pdbqt(text: str, type_names, pair_coeffs, solpar, vol) -> Ligand:
    """One ligand.  `type_names`: the atom-type names in map order (index = map index); the force-field tables
    (pair_coeffs [T][T][4], solpar [T], vol [T]) come from the caller.  Atom order = file order."""
    serial_to_idx, xyz, charge, types = {}, [], [], []
    rot, bonds, in_root, root_atom = [], [], False, None
    tindex = {n.upper(): i for i, n in enumerate(type_names)}
    for ln in text.splitlines():
        rec = ln[:6].strip()
        if rec in ("ATOM", "HETATM"):
            serial = int(ln[6:11])
            serial_to_idx[serial] = len(xyz)
            xyz.append((float(ln[30:38]), float(ln[38:46]), float(ln[46:54])))
            charge.append(float(ln[66:76]))
            at = ln[77:79].strip().upper()
            if at not in tindex:
                raise ValueError(f"atom type {at!r} of atom {serial} has no map (known: {list(type_names)})")
            types.append(tindex[at])
            if in_root and root_atom is None:
                root_atom = len(xyz) - 1
        elif rec == "ROOT":
            in_root = True
        elif rec == "ENDROO":
            in_root = False
        elif rec == "BRANCH":
            a, b = ln.split()[1:3]
            rot.append((int(a), int(b)))
        elif rec == "CONECT":
            f = [int(ln[6 + 5 * k:11 + 5 * k]) for k in range((len(ln.rstrip()) - 6 + 4) // 5)]
            bonds += [(f[0], o) for o in f[1:]]
    if not xyz:
        raise ValueError("no ATOM / HETATM records")
    X = np.array(xyz, np.float32)
    n = len(xyz)
    try:
        rot_idx = np.array([(serial_to_idx[a], serial_to_idx[b]) for a, b in rot], np.int32).reshape(-1, 2)
        if bonds:
            bset = {tuple(sorted((serial_to_idx[a], serial_to_idx[b]))) for a, b in bonds}
        else:
            bset = None
    except KeyError as e:
        raise ValueError(f"BRANCH / CONECT names unknown atom serial {e.args[0]}") from None
    if bset is None:                                         # distance rule: d < 1.1 (r_i + r_j)
        names = [type_names[t] for t in types]
        r = np.array([_COVALENT.get(_element(a), 0.76) for a in names])
        d = np.linalg.norm(X[:, None, :].astype(np.float64) - X[None, :, :], axis=-1)
        i, j = np.nonzero(np.triu(d < 1.1 * (r[:, None] + r[None, :]), 1))
        bset = set(zip(i.tolist(), j.tolist()))
    bset |= {tuple(sorted(map(int, p))) for p in rot_idx}    # a BRANCH is a bond
    B = np.array(sorted(bset), np.int32).reshape(-1, 2)
    return Ligand(X, np.array(types, np.int32), np.array(charge, np.float32), B, rot_idx, int(root_atom or 0), len(type_names),
                  np.asarray(pair_coeffs, np.float32), np.asarray(solpar, np.float32), np.asarray(vol, np.float32))


def write_pdbqt(lig: Ligand, type_names, conect: bool = True):
    """PDBQT text of `lig` (ROOT block, nested BRANCH blocks) and the atom order it was written in (file atom k =
    lig atom order[k]).  Used by the tests to round-trip synthetic ligands; CONECT records carry the bonds."""
    n = lig.N
    rot = {tuple(sorted(map(int, p))) for p in lig.rot_bonds}
    adj = [[] for _ in range(n)]
    for a, b in lig.bonds.tolist():
        adj[a].append(b); adj[b].append(a)
    frag = [-1] * n
    def flood(start, f):
        stack = [start]; frag[start] = f
        while stack:
            u = stack.pop()
            for v in adj[u]:
                if frag[v] < 0 and tuple(sorted((u, v))) not in rot:
                    frag[v] = f; stack.append(v)
    nf = 0
    for i in range(n):
        if frag[i] < 0:
            flood(i, nf); nf += 1
    order, lines, serial = [], [], {}
    def atom_line(i):
        serial[i] = len(order) + 1
        order.append(i)
        x, y, z = (float(v) for v in lig.xyz[i])
        return (f"{'ATOM':<6}{serial[i]:>5} {'C':<4} {'LIG':>3} {'A':>1}{1:>4}    {x:8.3f}{y:8.3f}{z:8.3f}{1.0:6.2f}{0.0:6.2f}"
                f"{float(lig.charge[i]):10.3f} {type_names[int(lig.type[i])]:<2}")
    done = set()
    root_f = frag[lig.root_atom]
    def emit(f, first):                                      # `first`: the atom written first (root atom / b of the branch)
        done.add(f)
        members = [first] + [i for i in range(n) if frag[i] == f and i != first]
        for i in members:
            lines.append(atom_line(i))
        if f == root_f:
            lines.append("ENDROOT")
        for i in members:
            for v in adj[i]:
                if frag[v] not in done and tuple(sorted((i, v))) in rot:
                    lines.append(f"BRANCH {serial[i]:>3} {len(order) + 1:>3}")
                    emit(frag[v], v)
                    lines.append(f"ENDBRANCH {serial[i]:>3} {serial[v]:>3}")
    lines.append("ROOT")
    emit(root_f, lig.root_atom)
    if conect:
        for a, b in lig.bonds.tolist():
            lines.append(f"CONECT{serial[a]:>5}{serial[b]:>5}")
    lines.append(f"TORSDOF {len(rot)}")
    return "\n".join(lines) + "\n", order


def write_map(values: np.ndarray, spacing: float, origin) -> str:
    """AutoGrid .map text of one map [nz][ny][nx] (x fastest); CENTER = origin + spacing * (n-1)/2"""
    nz, ny, nx = values.shape
    c = np.asarray(origin, np.float64) + 0.5 * spacing * np.array([nx - 1, ny - 1, nz - 1])
    head = ["GRID_PARAMETER_FILE synthetic.gpf", "GRID_DATA_FILE synthetic.maps.fld", "MACROMOLECULE synthetic.pdbqt",
            f"SPACING {spacing:.6f}", f"NELEMENTS {nx - 1} {ny - 1} {nz - 1}", f"CENTER {c[0]:.6f} {c[1]:.6f} {c[2]:.6f}"]
    return "\n".join(head + [f"{v:.9g}" for v in values.reshape(-1)]) + "\n"


def read_maps(texts) -> GridSet:
    """texts: the .map files in map order (atom types..., electrostatic, desolvation); all must share one geometry."""
    maps, geom = [], None
    for t in texts:
        ls = t.splitlines()
        hdr = {l.split()[0]: l.split()[1:] for l in ls[:6]}
        try:
            h = float(hdr["SPACING"][0])
            e = tuple(int(v) for v in hdr["NELEMENTS"])
            c = tuple(float(v) for v in hdr["CENTER"])
        except (KeyError, IndexError, ValueError):
            raise ValueError("map header needs SPACING, NELEMENTS and CENTER in its first 6 lines") from None
        nx, ny, nz = e[0] + 1, e[1] + 1, e[2] + 1
        vals = np.array([float(v) for v in ls[6:6 + nx * ny * nz]], np.float32)
        if vals.size != nx * ny * nz:
            raise ValueError(f"map holds {vals.size} values, NELEMENTS asks for {nx * ny * nz}")
        if geom is None:
            geom = (h, e, c)
        elif geom != (h, e, c):
            raise ValueError("maps differ in SPACING / NELEMENTS / CENTER")
        maps.append(vals.reshape(nz, ny, nx))
    h, e, c = geom
    origin = np.array([c[k] - 0.5 * h * e[k] for k in range(3)], np.float32)
    return GridSet(np.stack(maps), h, origin, {"source": "autogrid maps"})
