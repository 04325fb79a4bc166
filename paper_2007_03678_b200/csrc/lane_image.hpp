// lane_image.hpp -- ligand image for the lane-per-individual kernels (lane.cuh).
// One THREAD evaluates one genotype; the 32 lanes of a warp hold 32 genotypes of the same ligand, so everything
// in this image is warp-uniform and is read from shared memory by broadcast.  Atoms are renumbered in fragment
// DFS preorder ("lane order"): every rigid fragment is a contiguous range and parents precede children.
// The non-excluded pair list (R2) is cut into register tiles: an I-block of kLaneBI consecutive atoms
// (kept in registers with their force accumulators) against one aligned J-pair (atoms 2m, 2m+1: the two halves
// of a packed f32x2 operand).  A tile is evaluated as two HALVES of two rows (rows 0-1, rows 2-3): the two rows of a
// half are independent dependency chains issued in one basic block.  A tile lists only its active halves; a slot
// whose pair is excluded (including a whole row of an active half) carries zero coefficients and contributes
// exactly zero.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#include "topology.hpp"

namespace adock {

#ifndef ADOCK_LANE_BI
#define ADOCK_LANE_BI 4
#endif
constexpr int kLaneBI = ADOCK_LANE_BI;      // rows (I atoms) per register block: 4 or 8
constexpr int kLaneParts = 4;   // the tile sequence is cut into this many runs of (nearly) equal row count, so that
                                // K = 1, 2 or 4 warps can share the pair work of the same 32 individuals (lane.cuh)

struct LaneHeader {             // 128 bytes
    int N, Npad, R, nfrag;      // Npad = N rounded up to a multiple of kLaneBI (pad atoms sit at the origin, in no pair)
    int nblocks, ntiles, nrows, maxdepth;
    int off_atoms, off_types, off_frags, off_blocks;    // types: cell set (2 type + (q < 0)) | fragment << 8 per atom, -1 = pad
    int off_tiles, off_rows, bytes, npairs;
    int own_floats, warp_floats, nslots, own_a; // per-thread scratch: own_a float4 (4 sums per fragment) + nfrag float2 (2 sums):
                                                // own_floats = 4 own_a + 2 nfrag >= 12 maxdepth (the transform stack of the pose);
                                                // warp_floats = 3 Npad + own_floats + (7+R)  (one warp per group)
    int part_blk[kLaneParts + 1];               // part p owns blocks [part_blk[p], part_blk[p+1])
    int part_row[kLaneParts + 1];               // and row records from part_row[p] on (a block may be cut between parts)
    int pad2[2];
};
static_assert(kLaneBI == 4 || kLaneBI == 8, "kLaneBI");
static_assert(sizeof(LaneHeader) == 128, "LaneHeader layout");
struct LaneFrag {               // 48 bytes; fragments in DFS preorder
    int parent;                 // -1 for the root
    int depth_kids;             // depth (root 0) | has_children << 16
    int abeg, aend;             // atoms [abeg,aend) in lane order
    float p0[3]; int tor;       // x0[a_k] - pivot ; caller's torsion index (-1 for the root)
    float u[3];  int ab;        // unit(x0[b_k] - x0[a_k]) ; lane position of a_k | lane position of b_k << 16
};
struct LaneBlock {              // 32 bytes: I atoms kLaneBI*b .. kLaneBI*b + kLaneBI-1 of an active block
    int b;                      // block index
    int tile_begin, tile_end;
    int pad0;
    uint32_t frags[2];          // fragment id of row r in byte r&3 of frags[r>>2]
    int pad1[2];
};
static_assert(sizeof(LaneBlock) == 32, "LaneBlock layout");
struct LaneTile {               // 8 bytes
    uint32_t w0;                // jp | halfmask << 8 (bit h: rows 2h, 2h+1) | half-has-12-10-slot << 12 ;
                                // each active half owns two consecutive row records, consumed in sequence
    uint32_t w1;                // hbmask (bit 2r+h) | frag(j0) << 16 | frag(j1) << 24
};
struct LaneRow {                // 32 bytes: one active row against the two J atoms (h = 0, 1)
    float c12[2], ncA[2];       // c12, -cA   (weighted coefficients, R5)
    float ds[2], qq[2];         // w_desolv (S_i V_j + S_j V_i) ; elec_scale q_i q_j
};

struct LaneImage {
    std::vector<unsigned char> blob;
    std::vector<int> pos_of_ext, ext_of_pos;    // [N], [Npad] (-1 = pad)
    int warp_floats = 0, npad = 0, own_floats = 0;
};

inline void build_lane_image(LaneImage& im, const Topology& tp, const float* xyz, const int* type, const float* charge,
                             const float* coeffs, const float* solpar, const float* vol, float w_desolv, float qasp,
                             double elec_scale) {       // elec_scale: already divided by the fold factor of pair_row (adock.cu)
    const int N = tp.N, R = tp.R, T = tp.T, nfrag = tp.nfrag;
    const int Npad = (N + kLaneBI - 1) / kLaneBI * kLaneBI;
    im.pos_of_ext.assign(N, -1);
    im.ext_of_pos.assign(Npad, -1);
    std::vector<int> abeg(nfrag), aend(nfrag), depth(nfrag, 0), kids(nfrag, 0), frag_of_pos(Npad, 0);
    int p = 0, maxdepth = 0;
    for (int f = 0; f < nfrag; ++f) {
        abeg[f] = p;
        for (int e : tp.frag_info[f].atoms) { im.pos_of_ext[e] = p; im.ext_of_pos[p] = e; frag_of_pos[p] = f; ++p; }
        aend[f] = p;
        const int par = tp.frag_info[f].parent;
        if (par >= 0) { depth[f] = depth[par] + 1; kids[par] = 1; }
        maxdepth = std::max(maxdepth, depth[f]);
    }
    // ---- tiles
    const int nblk_all = Npad / kLaneBI, njp = Npad / 2;
    struct Slot { bool on = false; int ei = 0, ej = 0; };
    std::vector<Slot> grid((size_t)Npad * Npad);
    for (size_t k = 0; k < tp.pairs.size(); k += 2) {
        const int a = im.pos_of_ext[tp.pairs[k]], b = im.pos_of_ext[tp.pairs[k + 1]];
        const int I = std::min(a, b), J = std::max(a, b);
        grid[(size_t)I * Npad + J] = {true, im.ext_of_pos[I], im.ext_of_pos[J]};
    }
    std::vector<LaneBlock> blocks;
    std::vector<LaneTile> tiles;
    std::vector<LaneRow> rows;
    int npair_slots = 0;
    for (int b = 0; b < nblk_all; ++b) {
        LaneBlock blk{};
        blk.b = b; blk.tile_begin = (int)tiles.size();
        for (int r = 0; r < kLaneBI; ++r) blk.frags[r >> 2] |= (uint32_t)frag_of_pos[b * kLaneBI + r] << (8 * (r & 3));
        for (int jp = 0; jp < njp; ++jp) {
            uint32_t halfmask = 0, hbmask = 0, hbhalf = 0;
            LaneRow trow[kLaneBI];
            for (int r = 0; r < kLaneBI; ++r) {
                const int I = b * kLaneBI + r;
                LaneRow row{};
                bool any = false;
                for (int h = 0; h < 2; ++h) {
                    const Slot& s = grid[(size_t)I * Npad + 2 * jp + h];
                    if (!s.on) continue;
                    any = true;
                    const int ti = type[s.ei], tj = type[s.ej];
                    const float* co = coeffs + ((size_t)ti * T + tj) * 4;
                    const double Si = (double)solpar[ti] + (double)qasp * std::fabs((double)charge[s.ei]);
                    const double Sj = (double)solpar[tj] + (double)qasp * std::fabs((double)charge[s.ej]);
                    row.c12[h] = co[0];
                    row.ncA[h] = -co[1];
                    row.ds[h] = (float)((double)w_desolv * (Si * (double)vol[tj] + Sj * (double)vol[ti]));
                    row.qq[h] = (float)(elec_scale * (double)charge[s.ei] * (double)charge[s.ej]);
                    if (co[2] > 8.0f) { hbmask |= 1u << (2 * r + h); hbhalf |= 1u << (r / 2); }
                    ++npair_slots;
                }
                trow[r] = row;
                if (any) halfmask |= 1u << (r / 2);
            }
            if (!halfmask) continue;
            for (int hf = 0; hf < kLaneBI / 2; ++hf)
                if (halfmask & (1u << hf)) { rows.push_back(trow[2 * hf]); rows.push_back(trow[2 * hf + 1]); }
            LaneTile t;
            t.w0 = (uint32_t)jp | (halfmask << 8) | (hbhalf << 12);
            t.w1 = hbmask | ((uint32_t)frag_of_pos[2 * jp] << 16) | ((uint32_t)frag_of_pos[2 * jp + 1] << 24);
            tiles.push_back(t);
        }
        blk.tile_end = (int)tiles.size();
        if (blk.tile_end > blk.tile_begin) blocks.push_back(blk);
    }
    // ---- parts: cut the tile sequence where the running row count crosses p/kLaneParts of the total
    int part_blk[kLaneParts + 1], part_row[kLaneParts + 1];
    {
        auto tile_rows = [&](int t) { const uint32_t hm = (tiles[t].w0 >> 8) & 15u; return 2 * (int)((hm & 1u) + ((hm >> 1) & 1u) + ((hm >> 2) & 1u) + (hm >> 3)); };
        const int total = (int)rows.size();
        std::vector<LaneBlock> cut;
        int p = 0, acc = 0;
        part_blk[0] = 0; part_row[0] = 0;
        for (const LaneBlock& b : blocks) {
            LaneBlock cur = b;
            for (int t = b.tile_begin; t < b.tile_end; ++t) {
                // a tile starts the next part when the rows before it reach the part's share
                while (p + 1 < kLaneParts && acc >= (long long)total * (p + 1) / kLaneParts && acc > part_row[p]) {
                    if (t > cur.tile_begin) { LaneBlock head = cur; head.tile_end = t; cut.push_back(head); cur.tile_begin = t; }
                    ++p;
                    part_blk[p] = (int)cut.size(); part_row[p] = acc;
                }
                acc += tile_rows(t);
            }
            cut.push_back(cur);
        }
        while (p < kLaneParts) { ++p; part_blk[p] = (int)cut.size(); part_row[p] = acc; }
        blocks.swap(cut);
    }
    // ---- blob
    auto align16 = [](size_t x) { return (x + 15) & ~(size_t)15; };
    LaneHeader h{};
    h.N = N; h.Npad = Npad; h.R = R; h.nfrag = nfrag;
    h.nblocks = (int)blocks.size(); h.ntiles = (int)tiles.size(); h.nrows = (int)rows.size(); h.maxdepth = maxdepth;
    h.npairs = (int)tp.pairs.size() / 2;
    h.own_a = std::max(nfrag, (12 * maxdepth - 2 * nfrag + 3) / 4);     // the stack (12 floats per depth) may run on into the float2 part
    h.own_floats = 4 * h.own_a + 2 * nfrag;
    h.warp_floats = 3 * Npad + h.own_floats + 7 + R;
    for (int q = 0; q <= kLaneParts; ++q) { h.part_blk[q] = part_blk[q]; h.part_row[q] = part_row[q]; }
    size_t off = sizeof(LaneHeader);
    h.off_atoms = (int)off;  off = align16(off + (size_t)Npad * 16);
    h.off_types = (int)off;  off = align16(off + (size_t)Npad * 4);
    h.off_frags = (int)off;  off = align16(off + (size_t)nfrag * sizeof(LaneFrag));
    h.off_blocks = (int)off; off = align16(off + blocks.size() * (sizeof(LaneBlock) + 0));
    h.off_tiles = (int)off;  off = align16(off + (tiles.size() + 1) * sizeof(LaneTile));    // + a sentinel (J-pair 0, no half):
                                                                                          // the tile loop reads one record ahead
    h.off_rows = (int)off;   off = align16(off + rows.size() * sizeof(LaneRow));
    h.bytes = (int)off;
    h.nslots = 2 * (int)rows.size();    // pair slots evaluated; npairs of them carry a pair
    (void)npair_slots;
    im.warp_floats = h.warp_floats; im.npad = Npad; im.own_floats = h.own_floats;
    im.blob.assign(off, 0);
    std::memcpy(im.blob.data(), &h, sizeof(h));
    float* atoms = (float*)(im.blob.data() + h.off_atoms);
    int* types = (int*)(im.blob.data() + h.off_types);
    for (int q = 0; q < Npad; ++q) {
        const int e = im.ext_of_pos[q];
        if (e < 0) { types[q] = -1; continue; }            // pad
        for (int d = 0; d < 3; ++d) atoms[4 * q + d] = (float)((double)xyz[3 * e + d] - (double)tp.pivot[d]);
        atoms[4 * q + 3] = charge[e];
        types[q] = (2 * type[e] + (charge[e] < 0.f ? 1 : 0)) | (frag_of_pos[q] << 8);       // cell set (device.cuh, grid term)
    }
    LaneFrag* fr = (LaneFrag*)(im.blob.data() + h.off_frags);
    for (int f = 0; f < nfrag; ++f) {
        fr[f].parent = tp.frag_info[f].parent;
        fr[f].depth_kids = depth[f] | (kids[f] << 16);
        fr[f].abeg = abeg[f]; fr[f].aend = aend[f];
        fr[f].tor = tp.frag_info[f].tor;
        if (fr[f].tor >= 0) {
            const int a = tp.rot[2 * fr[f].tor], b = tp.rot[2 * fr[f].tor + 1];
            double u[3], n = 0;
            for (int d = 0; d < 3; ++d) { u[d] = (double)xyz[3 * b + d] - (double)xyz[3 * a + d]; n += u[d] * u[d]; }
            n = std::sqrt(n);
            for (int d = 0; d < 3; ++d) {
                fr[f].p0[d] = (float)((double)xyz[3 * a + d] - (double)tp.pivot[d]);
                fr[f].u[d] = (float)(u[d] / n);
            }
            fr[f].ab = im.pos_of_ext[a] | (im.pos_of_ext[b] << 16);
        }
    }
    LaneBlock* bl = (LaneBlock*)(im.blob.data() + h.off_blocks);
    for (size_t k = 0; k < blocks.size(); ++k) bl[k] = blocks[k];
    if (!tiles.empty()) std::memcpy(im.blob.data() + h.off_tiles, tiles.data(), tiles.size() * sizeof(LaneTile));
    if (!rows.empty()) std::memcpy(im.blob.data() + h.off_rows, rows.data(), rows.size() * sizeof(LaneRow));
}

}  // namespace adock
