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
struct LigHeader {          // 64 bytes
    int N, R, nfrag, npairs;
    int nrounds, T, off_atoms, off_meta;
    int off_frag, off_fragidx, off_pairs, bytes;
    int max_frag_atoms, max_depth, pad0, pad1;
};
struct FragGeom {           // 32 bytes: torsion axis of the bond that attaches fragment f to its parent
    float p0[3]; float pad0;   // x0[a_k] - pivot
    float u0[3]; float pad1;   // unit(x0[b_k] - x0[a_k])
};
struct FragIdx {            // 16 bytes
    int parent;             // parent fragment (internal id); -1 for the root
    int atom_begin, atom_end;   // internal atom range of this fragment
    int sub_end_tor;        // (subtree end fragment id) | (external torsion index << 16); root: tor = 0xffff
};
struct PairRec {            // 16 bytes: one slot of a warp round
    uint32_t ij;            // i | j<<8 | hbond<<16 | valid<<17   (internal atom ids)
    float c12, cA, ds;      // weighted coefficients; ds = w_desolv*(S_i V_j + S_j V_i)
};

struct Topology {
    int N = 0, R = 0, T = 0, nfrag = 0;
    // canonical (external numbering)
    std::vector<int> pairs;               // [np][2]
    std::vector<int> tor_order, rot;      // [R], [R][2] oriented
    std::vector<unsigned char> moved;     // [R][N]
    std::vector<int> depth;
    float pivot[3] = {0, 0, 0};
    // internal numbering
    std::vector<int> ext_of_int, int_of_ext;
    std::vector<unsigned char> blob;      // device image
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

    // ---- internal numbering: fragments in DFS preorder (children by torsion index), atoms by fragment
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
    tp.ext_of_int.clear(); tp.int_of_ext.assign(N, -1);
    std::vector<int> fbeg(tp.nfrag), fend(tp.nfrag);
    int max_frag_atoms = 0;
    for (int f = 0; f < tp.nfrag; ++f) {
        fbeg[f] = (int)tp.ext_of_int.size();
        for (int e : frags[f].atoms) { tp.int_of_ext[e] = (int)tp.ext_of_int.size(); tp.ext_of_int.push_back(e); }
        fend[f] = (int)tp.ext_of_int.size();
        max_frag_atoms = std::max(max_frag_atoms, fend[f] - fbeg[f]);
    }

    // ---- pair schedule: rounds of 32 slots, every atom at most once as i and once as j per round
    struct P { int a, b; };
    std::vector<P> rem;
    for (size_t p = 0; p < tp.pairs.size(); p += 2) rem.push_back({tp.int_of_ext[tp.pairs[p]], tp.int_of_ext[tp.pairs[p + 1]]});
    std::vector<int> deg(N, 0);
    for (auto& p : rem) { ++deg[p.a]; ++deg[p.b]; }
    std::vector<PairRec> recs;
    auto make_rec = [&](int i, int j) {
        int ei = tp.ext_of_int[i], ej = tp.ext_of_int[j];
        int ti = type[ei], tj = type[ej];
        const float* co = coeffs + ((size_t)ti * T + tj) * 4;
        double Si = (double)solpar[ti] + (double)qasp * std::fabs((double)charge[ei]);
        double Sj = (double)solpar[tj] + (double)qasp * std::fabs((double)charge[ej]);
        PairRec r;
        r.ij = (uint32_t)i | ((uint32_t)j << 8) | ((co[2] > 8.0f ? 1u : 0u) << 16) | (1u << 17);
        r.c12 = co[0]; r.cA = co[1];
        r.ds = (float)((double)w_desolv * (Si * (double)vol[tj] + Sj * (double)vol[ti]));
        return r;
    };
    int nrounds = 0;
    while (!rem.empty()) {
        // highest remaining degree first, so crowded atoms are spread over the rounds
        std::stable_sort(rem.begin(), rem.end(), [&](const P& x, const P& y) {
            return std::max(deg[x.a], deg[x.b]) > std::max(deg[y.a], deg[y.b]);
        });
        AtomSet usedI, usedJ;
        std::vector<P> keep;
        int filled = 0;
        for (auto& p : rem) {
            if (filled < 32 && !usedI.test(p.a) && !usedJ.test(p.b)) {
                usedI.set(p.a); usedJ.set(p.b); recs.push_back(make_rec(p.a, p.b)); ++filled; --deg[p.a]; --deg[p.b];
            } else if (filled < 32 && !usedI.test(p.b) && !usedJ.test(p.a)) {
                usedI.set(p.b); usedJ.set(p.a); recs.push_back(make_rec(p.b, p.a)); ++filled; --deg[p.a]; --deg[p.b];
            } else {
                keep.push_back(p);
            }
        }
        for (; filled < 32; ++filled) recs.push_back(PairRec{0u, 0.f, 0.f, 0.f});
        rem.swap(keep);
        ++nrounds;
    }

    // ---- blob
    auto align16 = [](size_t x) { return (x + 15) & ~(size_t)15; };
    LigHeader h{};
    h.N = N; h.R = R; h.nfrag = tp.nfrag; h.npairs = (int)tp.pairs.size() / 2; h.nrounds = nrounds; h.T = T;
    size_t off = sizeof(LigHeader);
    h.off_atoms = (int)off;   off = align16(off + (size_t)N * 16);
    h.off_meta = (int)off;    off = align16(off + (size_t)N * 4);
    h.off_frag = (int)off;    off = align16(off + (size_t)tp.nfrag * sizeof(FragGeom));
    h.off_fragidx = (int)off; off = align16(off + (size_t)tp.nfrag * sizeof(FragIdx));
    h.off_pairs = (int)off;   off = align16(off + recs.size() * sizeof(PairRec));
    h.bytes = (int)off;
    h.max_frag_atoms = max_frag_atoms;
    int maxd = 0;
    for (int k = 0; k < R; ++k) maxd = std::max(maxd, tp.depth[k]);
    h.max_depth = maxd;
    tp.blob.assign(off, 0);
    std::memcpy(tp.blob.data(), &h, sizeof(h));
    float* atoms = (float*)(tp.blob.data() + h.off_atoms);
    uint32_t* meta = (uint32_t*)(tp.blob.data() + h.off_meta);
    for (int i = 0; i < N; ++i) {
        int e = tp.ext_of_int[i];
        for (int d = 0; d < 3; ++d) atoms[4 * i + d] = (float)((double)xyz[3 * e + d] - (double)tp.pivot[d]);
        atoms[4 * i + 3] = charge[e];
        meta[i] = (uint32_t)type[e] | ((uint32_t)frag_of[e] << 8);
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
    if (!recs.empty()) std::memcpy(tp.blob.data() + h.off_pairs, recs.data(), recs.size() * sizeof(PairRec));
    return true;
}

}  // namespace adock
