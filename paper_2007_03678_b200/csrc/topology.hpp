// topology.hpp -- host-side ligand preprocessing for the CUDA path (R2).
// Second, independent implementation of the integer structure (the oracle has its own): adjacency
// lists + bitsets instead of edge scans.  Produces (1) the canonical arrays exported through
// adock_ligand_pairs / adock_ligand_tree and (2) the device blob: atoms renumbered so every rigid
// fragment and every torsion subtree is a contiguous range, and the pair list packed into warp rounds in
// which no atom appears twice on the same side, so force scatter needs no atomics and is deterministic.
#pragma once
#include <algorithm>
#include <bitset>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <functional>
#include <string>
#include <vector>

namespace adock {

constexpr int kMaxAtoms = 256;
constexpr int kMaxTors = 64;
using AtomSet = std::bitset<kMaxAtoms>;

// ---- device blob layout (all sections 16-byte aligned; staged into shared memory in one bulk copy)
struct LigHeader {          // 80 bytes
    int N, R, nfrag, npairs;
    int nrounds, T, off_atoms, off_meta;
    int off_frag, off_fragidx, off_pairs, bytes;
    int max_frag_atoms, max_depth, npos, off_fragatoms;   // npos = 32*ceil(N/32) atom positions (some may be holes)
    int nfull, systolic, pad2, pad3;                      // rounds [0,nfull) have all 32 slots valid; systolic: see the pair schedule
};
struct FragGeom {           // 32 bytes: torsion axis of the bond that attaches fragment f to its parent
    float p0[3]; float pad0;   // x0[a_k] - pivot
    float u0[3]; float pad1;   // unit(x0[b_k] - x0[a_k])
};
struct FragIdx {            // 16 bytes
    int parent;             // parent fragment (internal id); -1 for the root
    int atom_begin, atom_end;   // this fragment's range in the fragatoms list (uint16 positions)
    int sub_end_tor;        // (subtree end fragment id) | (external torsion index << 16); root: tor = 0xffff
};
struct PairRec {            // 16 bytes: one slot of a warp round
    uint32_t ij;            // slot(i) | slot(j)<<11 | hbond<<22 | valid<<23, slot(q) = (q>>5)*256 + (q&31):
                            // word offset of the atom at position q in the per-warp pose block (device.cuh)
    float c12, cA, ds;      // weighted coefficients; ds = w_desolv*(S_i V_j + S_j V_i)
};
inline uint32_t atom_slot(int a) { return (uint32_t)((a >> 5) * 256 + (a & 31)); }

struct Topology {
    int N = 0, R = 0, T = 0, nfrag = 0;
    // canonical (external numbering)
    std::vector<int> pairs;               // [np][2]
    std::vector<int> tor_order, rot;      // [R], [R][2] oriented
    std::vector<unsigned char> moved;     // [R][N]
    std::vector<int> depth;
    float pivot[3] = {0, 0, 0};
    // positions: int_of_ext [N] atom -> position, ext_of_int [npos] position -> atom or -1 (hole)
    std::vector<int> ext_of_int, int_of_ext;
    std::vector<unsigned char> blob;      // device image
    // rigid fragments in DFS preorder (parent < child; a torsion's subtree is the range [f, sub_end)); tor = caller's
    // torsion index of the bond that attaches the fragment to its parent (-1 for the root); atoms in caller order
    struct FragInfo { int parent, tor, sub_end; std::vector<int> atoms; };
    std::vector<FragInfo> frag_info;
    std::vector<int> frag_of_ext;         // [N]
    std::string error;
};

inline bool build_topology(Topology& tp, int N, const float* xyz, const int* type, const float* charge, int nbonds,
                           const int* bonds, int R, const int* rot_in, int root, int T, const float* coeffs,
                           const float* solpar, const float* vol, float w_desolv, float qasp) {
    tp.N = N; tp.R = R; tp.T = T;
    std::vector<std::vector<int>> adj(N);
    for (int b = 0; b < nbonds; ++b) {
        int p = bonds[2 * b], q = bonds[2 * b + 1];
        if (p < 0 || q < 0 || p >= N || q >= N || p == q) { tp.error = "bond index out of range"; return false; }
        adj[p].push_back(q); adj[q].push_back(p);
    }
    auto flood = [&](int start, int ba, int bb, bool cut_rot) {
        // atoms reachable from start without crossing bond (ba,bb) [and without crossing any rotatable bond]
        AtomSet seen;
        std::vector<int> stack{start};
        seen.set(start);
        while (!stack.empty()) {
            int u = stack.back(); stack.pop_back();
            for (int v : adj[u]) {
                if ((u == ba && v == bb) || (u == bb && v == ba)) continue;
                if (cut_rot) {
                    bool is_rot = false;
                    for (int k = 0; k < R; ++k)
                        if ((rot_in[2 * k] == u && rot_in[2 * k + 1] == v) || (rot_in[2 * k] == v && rot_in[2 * k + 1] == u)) is_rot = true;
                    if (is_rot) continue;
                }
                if (!seen.test(v)) { seen.set(v); stack.push_back(v); }
            }
        }
        return seen;
    };
    // orientation and moved sets
    std::vector<AtomSet> mv(R);
    tp.rot.resize(2 * R); tp.depth.assign(R, 0);
    for (int k = 0; k < R; ++k) {
        int a = rot_in[2 * k], b = rot_in[2 * k + 1];
        if (a < 0 || b < 0 || a >= N || b >= N) { tp.error = "rotatable bond index out of range"; return false; }
        if (std::find(adj[a].begin(), adj[a].end(), b) == adj[a].end()) { tp.error = "rotatable bond is not a bond"; return false; }
        AtomSet root_side = flood(root, a, b, false);
        if (root_side.test(a) && root_side.test(b)) { tp.error = "rotatable bond lies in a ring"; return false; }
        if (!root_side.test(a)) std::swap(a, b);
        tp.rot[2 * k] = a; tp.rot[2 * k + 1] = b;
        mv[k] = flood(b, a, b, false);
    }
    tp.moved.assign((size_t)R * N, 0);
    for (int k = 0; k < R; ++k)
        for (int i = 0; i < N; ++i) tp.moved[(size_t)k * N + i] = mv[k].test(i);
    for (int k = 0; k < R; ++k)
        for (int k2 = 0; k2 < R; ++k2) tp.depth[k] += mv[k2].test(tp.rot[2 * k + 1]);
    tp.tor_order.resize(R);
    for (int k = 0; k < R; ++k) tp.tor_order[k] = k;
    std::stable_sort(tp.tor_order.begin(), tp.tor_order.end(), [&](int x, int y) { return tp.depth[x] > tp.depth[y]; });
    // pivot: float64 mean rounded once
    for (int d = 0; d < 3; ++d) {
        double s = 0;
        for (int i = 0; i < N; ++i) s += (double)xyz[3 * i + d];
        tp.pivot[d] = (float)(s / N);
    }
    // topological distance up to 3 by neighbourhood expansion
    std::vector<AtomSet> near(N);
    for (int i = 0; i < N; ++i) {
        AtomSet cur; cur.set(i);
        near[i] = cur;
        for (int step = 0; step < 3; ++step) {
            AtomSet nxt;
            for (int u = 0; u < N; ++u) if (cur.test(u)) for (int v : adj[u]) nxt.set(v);
            near[i] |= nxt; cur = nxt;
        }
    }
    tp.pairs.clear();
    for (int i = 0; i < N; ++i)
        for (int j = i + 1; j < N; ++j) {
            if (near[i].test(j)) continue;
            bool flex = false;
            for (int k = 0; k < R && !flex; ++k) {
                int a = tp.rot[2 * k], b = tp.rot[2 * k + 1];
                if (mv[k].test(i) != mv[k].test(j) && i != a && i != b && j != a && j != b) flex = true;
            }
            if (flex) { tp.pairs.push_back(i); tp.pairs.push_back(j); }
        }

    // ---- fragments in DFS preorder (children by torsion index): every torsion subtree is a contiguous fragment range
    std::vector<int> frag_of(N, -1);
    struct Frag { int parent, tor; std::vector<int> atoms; int sub_end; };
    std::vector<Frag> frags;
    std::function<void(int, int, int)> visit = [&](int atom, int parent, int tor) {
        int f = (int)frags.size();
        frags.push_back({parent, tor, {}, 0});
        AtomSet members = flood(atom, -1, -1, true);
        for (int i = 0; i < N; ++i) if (members.test(i)) { frag_of[i] = f; frags[f].atoms.push_back(i); }
        for (int k = 0; k < R; ++k)                      // children: torsions whose a_k is in this fragment
            if (members.test(tp.rot[2 * k]) && frag_of[tp.rot[2 * k + 1]] < 0) visit(tp.rot[2 * k + 1], f, k);
        frags[f].sub_end = (int)frags.size();
    };
    visit(root, -1, -1);
    tp.nfrag = (int)frags.size();
    for (int i = 0; i < N; ++i)
        if (frag_of[i] < 0) { tp.error = "ligand graph is not connected"; return false; }
    tp.frag_of_ext = frag_of;
    tp.frag_info.clear();
    for (const Frag& f : frags) tp.frag_info.push_back({f.parent, f.tor, f.sub_end, f.atoms});
    // ---- atom positions.  Position q = pass*32 + lane is the atom's slot in every per-warp array, so its
    // shared-memory bank is q mod 32.  Crowded atoms (many pairs) get a bank of their own; when N > 32 the
    // atoms with the fewest pairs share banks (longest-processing-time assignment of pair counts to banks).
    std::vector<int> deg_ext(N, 0);
    for (size_t p = 0; p < tp.pairs.size(); ++p) ++deg_ext[tp.pairs[p]];
    const int npass = (N + 31) / 32, npos = npass * 32;
    std::vector<int> by_deg(N);
    for (int i = 0; i < N; ++i) by_deg[i] = i;
    std::stable_sort(by_deg.begin(), by_deg.end(), [&](int x, int y) { return deg_ext[x] > deg_ext[y]; });
    std::vector<int> bank_load(32, 0), bank_cnt(32, 0);
    tp.ext_of_int.assign(npos, -1); tp.int_of_ext.assign(N, -1);
    for (int e : by_deg) {
        int best = -1;
        for (int r = 0; r < 32; ++r)
            if (bank_cnt[r] < npass && (best < 0 || bank_load[r] < bank_load[best])) best = r;
        const int q = bank_cnt[best] * 32 + best;
        tp.int_of_ext[e] = q; tp.ext_of_int[q] = e;
        ++bank_cnt[best]; bank_load[best] += deg_ext[e];
    }
    // fragment member lists (positions), fragment by fragment
    std::vector<uint16_t> fragatoms;
    std::vector<int> fbeg(tp.nfrag), fend(tp.nfrag);
    int max_frag_atoms = 0;
    for (int f = 0; f < tp.nfrag; ++f) {
        fbeg[f] = (int)fragatoms.size();
        for (int e : frags[f].atoms) fragatoms.push_back((uint16_t)tp.int_of_ext[e]);
        fend[f] = (int)fragatoms.size();
        max_frag_atoms = std::max(max_frag_atoms, fend[f] - fbeg[f]);
    }

    // ---- pair schedule: rounds of 32 slots.  Hard rule (correctness of the atomics-free force scatter): within a
    // round no atom occurs twice as i or twice as j.  Soft rule (speed): the i positions of a round are distinct
    // modulo 32, and so are the j positions, so each side touches 32 different banks; a slot that cannot be
    // filled under the soft rule is filled under the hard rule alone (a 2-way conflict beats an extra round).
    struct P { int a, b; };
    std::vector<P> rem;
    for (size_t p = 0; p < tp.pairs.size(); p += 2) rem.push_back({tp.int_of_ext[tp.pairs[p]], tp.int_of_ext[tp.pairs[p + 1]]});
    std::vector<int> deg(npos, 0);
    for (auto& p : rem) { ++deg[p.a]; ++deg[p.b]; }
    std::vector<PairRec> recs;
    auto make_rec = [&](int i, int j) {
        int ei = tp.ext_of_int[i], ej = tp.ext_of_int[j];
        int ti = type[ei], tj = type[ej];
        const float* co = coeffs + ((size_t)ti * T + tj) * 4;
        double Si = (double)solpar[ti] + (double)qasp * std::fabs((double)charge[ei]);
        double Sj = (double)solpar[tj] + (double)qasp * std::fabs((double)charge[ej]);
        PairRec r;
        r.ij = atom_slot(i) | (atom_slot(j) << 11) | ((co[2] > 8.0f ? 1u : 0u) << 22) | (1u << 23);
        r.c12 = co[0]; r.cA = co[1];
        r.ds = (float)((double)w_desolv * (Si * (double)vol[tj] + Sj * (double)vol[ti]));
        return r;
    };
    int nrounds = 0, nfull = 0;
    // Systolic schedule for ligands of exactly four position blocks (97..128 atoms), where the list schedule above spends most
    // of its shared-memory bandwidth on loading both atoms and updating both forces of every pair: round k * 4 + b
    // (k = 0 .. npos/2 - 1, b = block) pairs position i = 32 b + lane with j = (i + k + 1) mod npos, so a lane keeps ONE atom i
    // for all its rounds (position and force sum in registers) and only the j side touches shared memory, conflict-free
    // (consecutive lanes, consecutive positions).  Every unordered pair {i, j} comes up exactly once (for k + 1 = npos/2
    // only from i < npos/2); excluded pairs and holes are slots with the valid bit clear.  The hard rule of the list
    // schedule holds as well (a round's i are distinct, and so are its j), so kernels that do not know the schedule run it as
    // nrounds padded rounds.
    const bool systolic = npos == 128;
    if (systolic) {
        std::vector<char> has((size_t)npos * npos, 0);
        for (auto& p : rem) has[(size_t)p.a * npos + p.b] = has[(size_t)p.b * npos + p.a] = 1;
        for (int k = 0; k < npos / 2; ++k)
            for (int b = 0; b < npos / 32; ++b)
                for (int l = 0; l < 32; ++l) {
                    const int i = 32 * b + l, j = (i + k + 1) % npos;
                    const bool valid = has[(size_t)i * npos + j] && (k + 1 < npos / 2 || i < npos / 2);
                    recs.push_back(valid ? make_rec(i, j) : PairRec{atom_slot(i) | (atom_slot(j) << 11), 0.f, 0.f, 0.f});
                }
        nrounds = (npos / 2) * (npos / 32);
        rem.clear();
    }
    while (!rem.empty()) {
        // highest remaining degree first, so crowded atoms are spread over the rounds
        std::stable_sort(rem.begin(), rem.end(), [&](const P& x, const P& y) {
            return std::max(deg[x.a], deg[x.b]) > std::max(deg[y.a], deg[y.b]);
        });
        AtomSet atomI, atomJ;
        std::bitset<32> bankI, bankJ;
        std::vector<char> taken(rem.size(), 0);
        int filled = 0;
        for (int pass = 0; pass < 2 && filled < 32; ++pass)          // pass 0: soft + hard rule, pass 1: hard rule only
            for (size_t k = 0; k < rem.size() && filled < 32; ++k) {
                if (taken[k]) continue;
                const P p = rem[k];
                auto fits = [&](int i, int j) {
                    if (atomI.test(i) || atomJ.test(j)) return false;
                    return pass == 1 || (!bankI.test(i & 31) && !bankJ.test(j & 31));
                };
                int i = -1, j = -1;
                if (fits(p.a, p.b)) { i = p.a; j = p.b; } else if (fits(p.b, p.a)) { i = p.b; j = p.a; }
                if (i < 0) continue;
                atomI.set(i); atomJ.set(j); bankI.set(i & 31); bankJ.set(j & 31);
                recs.push_back(make_rec(i, j));
                taken[k] = 1; ++filled; --deg[p.a]; --deg[p.b];
            }
        if (filled == 32) ++nfull;
        for (; filled < 32; ++filled) recs.push_back(PairRec{0u, 0.f, 0.f, 0.f});
        std::vector<P> keep;
        for (size_t k = 0; k < rem.size(); ++k) if (!taken[k]) keep.push_back(rem[k]);
        rem.swap(keep);
        ++nrounds;
    }

    if (!systolic) {    // full rounds first (their kernel loop carries no validity tests), padded rounds after
        std::vector<PairRec> full, part;
        for (int r = 0; r < nrounds; ++r) {
            bool all = true;
            for (int l = 0; l < 32; ++l) all = all && ((recs[(size_t)r * 32 + l].ij >> 23) & 1u);
            auto& dst = all ? full : part;
            dst.insert(dst.end(), recs.begin() + (size_t)r * 32, recs.begin() + (size_t)(r + 1) * 32);
        }
        full.insert(full.end(), part.begin(), part.end());
        recs.swap(full);
    }

    // ---- blob
    auto align16 = [](size_t x) { return (x + 15) & ~(size_t)15; };
    LigHeader h{};
    h.N = N; h.R = R; h.nfrag = tp.nfrag; h.npairs = (int)tp.pairs.size() / 2; h.nrounds = nrounds; h.T = T;
    h.npos = npos; h.nfull = nfull; h.systolic = systolic ? 1 : 0;
    size_t off = sizeof(LigHeader);
    h.off_atoms = (int)off;     off = align16(off + (size_t)npos * 16);
    h.off_meta = (int)off;      off = align16(off + (size_t)npos * 4);
    h.off_frag = (int)off;      off = align16(off + (size_t)tp.nfrag * sizeof(FragGeom));
    h.off_fragidx = (int)off;   off = align16(off + (size_t)tp.nfrag * sizeof(FragIdx));
    h.off_fragatoms = (int)off; off = align16(off + fragatoms.size() * sizeof(uint16_t));
    h.off_pairs = (int)off;     off = align16(off + recs.size() * sizeof(PairRec));
    h.bytes = (int)off;
    h.max_frag_atoms = max_frag_atoms;
    int maxd = 0;
    for (int k = 0; k < R; ++k) maxd = std::max(maxd, tp.depth[k]);
    h.max_depth = maxd;
    tp.blob.assign(off, 0);
    std::memcpy(tp.blob.data(), &h, sizeof(h));
    float* atoms = (float*)(tp.blob.data() + h.off_atoms);
    uint32_t* meta = (uint32_t*)(tp.blob.data() + h.off_meta);
    for (int q = 0; q < npos; ++q) {
        const int e = tp.ext_of_int[q];
        if (e < 0) { meta[q] = 0xffffffffu; continue; }          // hole
        for (int d = 0; d < 3; ++d) atoms[4 * q + d] = (float)((double)xyz[3 * e + d] - (double)tp.pivot[d]);
        atoms[4 * q + 3] = charge[e];
        meta[q] = (uint32_t)(2 * type[e] + (charge[e] < 0.f ? 1 : 0)) | ((uint32_t)frag_of[e] << 8);     // cell set | fragment
    }
    FragGeom* fg = (FragGeom*)(tp.blob.data() + h.off_frag);
    FragIdx* fi = (FragIdx*)(tp.blob.data() + h.off_fragidx);
    for (int f = 0; f < tp.nfrag; ++f) {
        fi[f].parent = frags[f].parent;
        fi[f].atom_begin = fbeg[f]; fi[f].atom_end = fend[f];
        int tor = frags[f].tor;
        fi[f].sub_end_tor = frags[f].sub_end | ((tor < 0 ? 0xffff : tor) << 16);
        if (tor >= 0) {
            int a = tp.rot[2 * tor], b = tp.rot[2 * tor + 1];
            double u[3], n = 0;
            for (int d = 0; d < 3; ++d) { u[d] = (double)xyz[3 * b + d] - (double)xyz[3 * a + d]; n += u[d] * u[d]; }
            n = std::sqrt(n);
            if (!(n > 1e-6)) { tp.error = "zero-length rotatable bond"; return false; }
            for (int d = 0; d < 3; ++d) {
                fg[f].p0[d] = (float)((double)xyz[3 * a + d] - (double)tp.pivot[d]);
                fg[f].u0[d] = (float)(u[d] / n);
            }
        }
    }
    if (!fragatoms.empty()) std::memcpy(tp.blob.data() + h.off_fragatoms, fragatoms.data(), fragatoms.size() * sizeof(uint16_t));
    if (!recs.empty()) std::memcpy(tp.blob.data() + h.off_pairs, recs.data(), recs.size() * sizeof(PairRec));
    return true;
}

}  // namespace adock
