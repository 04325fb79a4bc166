// lane.cuh -- lane-per-individual device code of the hot path.
// One LANE holds one genotype: pose (R3), grid term (R4), intramolecular pairs (R5), back-propagation (R6) and the
// ADADELTA chain (R7).  The 32 lanes of a warp hold 32 individuals of the SAME ligand, so the ligand image
// (lane_image.hpp) is read from shared memory by broadcast, control flow is warp-uniform, and no shuffle, atomic or
// cross-lane reduction is needed anywhere.  Per-lane state lives in shared memory as [index][lane] columns
// (conflict-free): atom positions relative to the translation, and per-fragment (force, torque) accumulators.
// A GROUP of K warps (K = 1, 2, 4) works on the same 32 individuals: the atoms of the grid phase and the parts of the
// pair-tile sequence are dealt out to the K warps, each accumulating into its own (force, torque) columns; part 0 adds
// them up and runs the serial tail.  More warps per individual = more warps per SM for the same shared memory (the
// positions are shared) and shorter chains.  The pair loop keeps an I-block of 4 atoms in registers and evaluates
// two rows at a time against an aligned J-pair with packed f32x2 arithmetic (FFMA2/FMUL2/FADD2).
// TM variants (one warp per group only) keep the atom positions in TENSOR MEMORY instead of shared memory: TMEM is
// 128 lanes x 512 columns of 32 bits per SM, a warp reaches the 32 lanes of its quarter with tcgen05.ld/st.32x32b, thread i
// <-> lane i, and the column address is warp-uniform -- exactly the [index][lane] access pattern of the per-lane state.
// Positions are 62 % of that state at 40 atoms; with them out of shared memory 12 or 16 warps per SM fit instead of 8.
#pragma once
#include "device.cuh"
#include "lane_image.hpp"

namespace adock {

// ---------------------------------------------------------------- tensor memory as per-lane scratch
// columns of one warp's slice when W warps share the 4 lane quarters
__host__ __device__ inline int lane_tmem_columns(int W) { return 512 / ((W + 3) / 4); }
__device__ __forceinline__ void tm_st1(uint32_t a, float v) { asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void tm_ld1(uint32_t a, float& v) { asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(v) : "r"(a) : "memory"); }
__device__ __forceinline__ void tm_ld2(uint32_t a, float& v0, float& v1) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(v0), "=f"(v1) : "r"(a) : "memory");
}
__device__ __forceinline__ void tm_ld4(uint32_t a, float& v0, float& v1, float& v2, float& v3) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=f"(v0), "=f"(v1), "=f"(v2), "=f"(v3) : "r"(a) : "memory");
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// The loaded registers are in/out operands of the wait, so no use of them can be scheduled ahead of it.
__device__ __forceinline__ void tm_wait_ld(float& a, float& b, float& c) { asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(a), "+f"(b), "+f"(c)::"memory"); }
__device__ __forceinline__ void tm_wait_ld(float& a, float& b, float& c, float& d, float& e, float& f) {
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(a), "+f"(b), "+f"(c), "+f"(d), "+f"(e), "+f"(f)::"memory");
}
__device__ __forceinline__ void tm_wait_ld(float& a, float& b, float& c, float& d, float& e, float& f, float& g, float& h, float& i,
                                           float& j, float& k, float& l) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+f"(a), "+f"(b), "+f"(c), "+f"(d), "+f"(e), "+f"(f), "+f"(g), "+f"(h), "+f"(i), "+f"(j), "+f"(k), "+f"(l)::"memory");
}
// All threads of the CTA call these.  open: one warp allocates all 512 columns (the kernels run one CTA per SM) and the
// address travels through the word at smem + 8 (behind the bulk-copy barrier); close: after every warp is done.
template <bool TM>
__device__ __forceinline__ uint32_t lane_tmem_open(unsigned char* smem) {
    if (!TM) return 0u;
    uint32_t* slot = reinterpret_cast<uint32_t*>(smem + 8);
    if ((threadIdx.x >> 5) == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *slot;
}
template <bool TM>
__device__ __forceinline__ void lane_tmem_close(uint32_t base) {
    if (!TM) return;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if ((threadIdx.x >> 5) == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}

// ---------------------------------------------------------------- views
struct LaneL {              // the staged image
    const float4* atoms;    // [Npad] x0 - pivot, q
    const int* types;       // [Npad] type, -1 = pad
    const int4* fragi;      // LaneFrag as 3 x 16 bytes
    const int4* blocks;
    const uint2* tiles;
    const float4* rows;
    int N, Npad, R, nfrag, nblocks, own_floats, own_a;
    const int* part_blk;    // [kLaneParts+1]
    const int* part_row;    // [kLaneParts+1]
};
__device__ inline LaneL lane_view(const unsigned char* blob) {
    const LaneHeader* h = reinterpret_cast<const LaneHeader*>(blob);
    LaneL L;
    L.atoms = reinterpret_cast<const float4*>(blob + h->off_atoms);
    L.types = reinterpret_cast<const int*>(blob + h->off_types);
    L.fragi = reinterpret_cast<const int4*>(blob + h->off_frags);
    L.blocks = reinterpret_cast<const int4*>(blob + h->off_blocks);
    L.tiles = reinterpret_cast<const uint2*>(blob + h->off_tiles);
    L.rows = reinterpret_cast<const float4*>(blob + h->off_rows);
    L.N = h->N; L.Npad = h->Npad; L.R = h->R; L.nfrag = h->nfrag; L.nblocks = h->nblocks; L.own_floats = h->own_floats; L.own_a = h->own_a;
    L.part_blk = h->part_blk; L.part_row = h->part_row;
    return L;
}
struct LaneS {              // this lane's columns of the group's scratch; element k of an array sits at [k*32]
    float2* P;              // [Npad/2][3]: positions RELATIVE TO t of atoms 2m (.x) and 2m+1 (.y): component c of pair m at
                            // P[(3m + c)*32] (one address register reaches x, y and z of a pair); unused by the TM variants
    uint32_t tp;            // TM variants: tensor-memory address (lane quarter | first column) of this warp's position
                            // columns: pair m at columns 6m .. 6m+5 = x0 x1 y0 y1 z0 z1
    float4* oA;             // per-fragment sums of THIS part, read and written as vectors: fragment f = (Fx, Fy, Fz, Tx) in
    float2* oB;             // oA[f*32] and (Ty, Tz) in oB[f*32] (force, torque about t); own_floats = 4 own_a + 2 nfrag floats.
                            // During the pose oA holds the transform stack: depth d = rows oA[(3d .. 3d+2)*32] of a 3x4 matrix
    int part_stride;        // floats between the own arrays of consecutive parts (own_floats*32); part 0's = this - part*stride
    float* geno;            // [7+R]
    float* ex;              // [8K+1]: (e_grid, e_pairs, grid force F(3), grid torque about t T(3)) of each part, then the
                            // chain's live flag
    float* state;           // ST: ADADELTA / Solis-Wets state columns of this lane: best [7+R], Eg2 [6+R], Ed2 [6+R]
    int part, gid;          // this warp's part in the group; group index in the CTA (named barrier gid+1)
};
// floats per lane of one group's shared-memory scratch (TM: the positions live in tensor memory)
// ST: the local-search state (best genotype and two accumulators per degree of freedom) sits in shared memory as well
__host__ __device__ inline int lane_group_floats(int Npad, int own_floats, int R, int K, bool TM = false, bool ST = false) {
    return (TM ? 0 : 3 * Npad) + K * own_floats + (7 + R) + (K > 1 ? 8 * K + 1 : 0)      // one warp per group exchanges nothing
           + (ST ? (7 + R) + 2 * (6 + R) : 0);
}
// group_floats = floats per lane between consecutive groups of the CTA: lane_group_floats of the ligand, or of the
// largest ligand of the launch when the groups of a CTA belong to different ligands (0 = this ligand's)
// tmem = lane_tmem_open's result (TM variants): warp w owns lanes 32 (w mod 4) and the (w / 4)-th slice of the 512 columns
template <int K, bool TM = false>
__device__ inline LaneS lane_scratch(float* cta_base, const LaneL& L, int warp, int lane, int group_floats = 0, uint32_t tmem = 0) {
    LaneS S;
    S.gid = warp / K; S.part = warp % K;
    if (group_floats == 0) group_floats = lane_group_floats(L.Npad, L.own_floats, L.R, K, TM);      // callers with ST pass it
    float* base = cta_base + (size_t)S.gid * group_floats * 32;
    S.P = reinterpret_cast<float2*>(base) + lane;
    S.tp = tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * lane_tmem_columns((int)(blockDim.x >> 5)));
    float* own = base + (TM ? 0 : 3 * L.Npad) * 32;   // 128-byte aligned
    S.part_stride = L.own_floats * 32;
    S.oA = reinterpret_cast<float4*>(own + S.part * S.part_stride) + lane;
    S.oB = reinterpret_cast<float2*>(own + S.part * S.part_stride + 4 * L.own_a * 32) + lane;
    S.geno = own + K * S.part_stride + lane;
    S.ex = S.geno + (7 + L.R) * 32;
    S.state = S.ex + (K > 1 ? 8 * K + 1 : 0) * 32;
    return S;
}
// barrier of the K warps of a group
template <int K>
__device__ __forceinline__ void group_sync(const LaneS& S) {
    if (K > 1) asm volatile("bar.sync %0, %1;" ::"r"(S.gid + 1), "r"(K * 32) : "memory");
}

// ---------------------------------------------------------------- atom positions (shared memory, or tensor memory when TM)
struct Pos6 { float x0, x1, y0, y1, z0, z1; };     // the J-pair (2m, 2m+1)
// issue the loads of pair m; pos_wait before the first use
template <bool TM>
__device__ __forceinline__ void pos_issue(const LaneS& S, int m, Pos6& p) {
    if (TM) {
        tm_ld4(S.tp + 6 * m, p.x0, p.x1, p.y0, p.y1);
        tm_ld2(S.tp + 6 * m + 4, p.z0, p.z1);
    } else {
        const float2* q = S.P + m * 96;
        const float2 a = q[0], b = q[32], c = q[64];
        p.x0 = a.x; p.x1 = a.y; p.y0 = b.x; p.y1 = b.y; p.z0 = c.x; p.z1 = c.y;
    }
}
template <bool TM> __device__ __forceinline__ void pos_wait(Pos6& p) { if (TM) tm_wait_ld(p.x0, p.x1, p.y0, p.y1, p.z0, p.z1); }
template <bool TM> __device__ __forceinline__ void pos_wait(Pos6& p, Pos6& q) {
    if (TM) tm_wait_ld(p.x0, p.x1, p.y0, p.y1, p.z0, p.z1, q.x0, q.x1, q.y0, q.y1, q.z0, q.z1);
}
// one atom
template <bool TM>
__device__ __forceinline__ void pos_put(const LaneS& S, int i, float x, float y, float z) {
    if (TM) {
        const uint32_t a = S.tp + 6 * (i >> 1) + (i & 1);
        tm_st1(a, x); tm_st1(a + 2, y); tm_st1(a + 4, z);
    } else {
        float* q = reinterpret_cast<float*>(S.P) + (i >> 1) * 192 + (i & 1);
        q[0] = x; q[64] = y; q[128] = z;
    }
}
template <bool TM>
__device__ __forceinline__ void pos_issue1(const LaneS& S, int i, float& x, float& y, float& z) {
    if (TM) {
        const uint32_t a = S.tp + 6 * (i >> 1) + (i & 1);
        tm_ld1(a, x); tm_ld1(a + 2, y); tm_ld1(a + 4, z);
    } else {
        const float* q = reinterpret_cast<const float*>(S.P) + (i >> 1) * 192 + (i & 1);
        x = q[0]; y = q[64]; z = q[128];
    }
}

// ---------------------------------------------------------------- one packed row of the pair tile (R5)
struct PairK {              // packed constants
    f2 k1, lk, one, A, B, k2, six, isig2;    // A, B: diel_A/s, diel_B/s (ParDev)
    float rmin2;
};
__device__ __forceinline__ PairK make_pairk(const ParDev& P) {
    PairK K;
    K.k1 = bc(P.mlamB_log2e); K.lk = bc(P.log2_dk); K.one = bc(1.f); K.A = bc(P.diel_As); K.B = bc(P.diel_Bs);
    K.k2 = bc(P.mhalf_inv_sig2_log2e); K.six = bc(6.f); K.isig2 = bc(P.inv_sig2);
    K.rmin2 = P.rmin2;
    return K;
}

// Row atom i (broadcast to both halves) against J atoms (j0 | j1).  Accumulates the pair energies into e2, and
// ns*d into BOTH gi (which therefore holds MINUS the gradient on i) and gj (the gradient on j), ns = -(dE/dr)/r.
template <bool GRAD, bool HB>
__device__ __forceinline__ void pair_row(const PairK& K, f2 xi, f2 yi, f2 zi, f2 xj, f2 yj, f2 zj, float4 ra, float4 rb,
                                         unsigned hb, f2& e2, f2& gix, f2& giy, f2& giz, f2& gjx, f2& gjy, f2& gjz) {
    const f2 dx = sub2(xi, xj), dy = sub2(yi, yj), dz = sub2(zi, zj);
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, mul2(dz, dz)));
    float r2l, r2h;
    unpk(r2, r2l, r2h);
    const float cl = fmaxf(r2l, K.rmin2), ch = fmaxf(r2h, K.rmin2);
    const f2 r2c = pk(cl, ch);
    const f2 rinv = pk(frsqrt(cl), frsqrt(ch));
    const f2 rr = mul2(r2c, rinv);
    const f2 rinv2 = mul2(rinv, rinv);
    const f2 rinv4 = mul2(rinv2, rinv2);
    const f2 r6 = mul2(rinv4, rinv2);
    const f2 c12 = pk(ra.x, ra.y), ncA = pk(ra.z, ra.w), ds = pk(rb.x, rb.y), qq = pk(rb.z, rb.w);
    const f2 u12 = mul2(mul2(c12, r6), r6);
    f2 rA = r6;
    if (HB) {                                   // 12-10 slot(s) in this half: rare
        float a, b, l, h;
        unpk(mul2(r6, rinv4), a, b);
        unpk(r6, l, h);
        rA = pk((hb & 1u) ? a : l, (hb & 2u) ? b : h);
    }
    const f2 evdw = fma2(ncA, rA, u12);          // c12 r^-12 - cA r^-A
    // electrostatics with the distance-dependent dielectric: eps = A + B/den, den = 1 + k exp(-lambda B r), and
    // k exp(-lambda B r) = 2^(-lambda B log2(e) r + log2 k): the factor k rides in the exponent
    float tl, th;
    unpk(fma2(rr, K.k1, K.lk), tl, th);
    const f2 kex = pk(fex2(tl), fex2(th));
    const f2 den = add2(kex, K.one);
    const f2 num = fma2(K.A, den, K.B);          // eps = s num/den, s = B lambda B
    unpk(mul2(den, num), tl, th);
    const f2 inv = pk(frcp(tl), frcp(th));       // s/(den eps den)
    const f2 ieps = mul2(mul2(den, den), inv);   // s/eps
    const f2 eel = mul2(mul2(qq, rinv), ieps);   // the row's qq carries 1/s
    // desolvation
    unpk(mul2(r2c, K.k2), tl, th);
    const f2 egs = mul2(ds, pk(fex2(tl), fex2(th)));
    e2 = add2(e2, add2(evdw, add2(eel, egs)));
    if (GRAD) {
        // -dE/dr = rinv (12 u12 - nA uA + eel) + eel (deps/dr)/eps + (r/sigma^2) egs ;  ns = -(dE/dr)/r
        const f2 s = add2(evdw, u12);
        f2 A1 = fma2(K.six, s, eel);
        if (HB) A1 = fma2(pk((hb & 1u) ? 4.f : 0.f, (hb & 2u) ? 4.f : 0.f), mul2(ncA, rA), A1);
        const f2 dee = mul2(kex, inv);              // (d eps/dr)/eps = B lambda B kex/(den^2 eps)
        const f2 A3 = fma2(eel, dee, mul2(A1, rinv));
        // desolvation: (r/sigma^2) egs / r = egs/sigma^2 (the clamped case is zeroed below)
        float nl, nh;
        unpk(fma2(A3, rinv, mul2(K.isig2, egs)), nl, nh);
        const f2 ns = pk(r2l >= K.rmin2 ? nl : 0.f, r2h >= K.rmin2 ? nh : 0.f);
        gix = fma2(ns, dx, gix); giy = fma2(ns, dy, giy); giz = fma2(ns, dz, giz);
        gjx = fma2(ns, dx, gjx); gjy = fma2(ns, dy, gjy); gjz = fma2(ns, dz, gjz);
    }
}

// own[f] += (F, T)
__device__ __forceinline__ void own_add(const LaneS& S, int f, float Fx, float Fy, float Fz, float Tx, float Ty, float Tz) {
    float4 a = S.oA[f * 32];
    float2 b = S.oB[f * 32];
    a.x += Fx; a.y += Fy; a.z += Fz; a.w += Tx; b.x += Ty; b.y += Tz;
    S.oA[f * 32] = a; S.oB[f * 32] = b;
}

// flush a fragment's (force, torque) sums: one warp per group visits every fragment exactly once (store); with K > 1 a
// part may skip fragments, so own[] is zeroed first and the sums are added
template <int K>
__device__ __forceinline__ void own_flush(const LaneS& S, int f, float Fx, float Fy, float Fz, float Tx, float Ty, float Tz) {
    if (K == 1) { S.oA[f * 32] = make_float4(Fx, Fy, Fz, Tx); S.oB[f * 32] = make_float2(Ty, Tz); }
    else own_add(S, f, Fx, Fy, Fz, Tx, Ty, Tz);
}

// ---------------------------------------------------------------- full evaluation of this lane's genotype
// Called by all K warps of the group with S.geno ready (and visible to all of them).  Part 0 returns the total energy
// (NaN for |q| < 1e-12, with NaN gradient); the other parts return 0.  With GRAD part 0 clears `gfin` if a gradient
// component is not finite and delivers the gradient according to GOUT:
//   GOUT = 1: grad[d*gs] for d < 6+R when `wr` (scoring: straight to the caller's array)
//   GOUT = 2: left in part 0's own[] columns: dE/dt, dE/domega in oA[0], oB[0], dE/dtau of fragment f's torsion in
//             oA[f*32].x (local search: the optimiser reads them from shared memory; `grad` is not used)
// The rigid-body blocks (dE/dt, dE/domega) are summed from the GRID forces alone: intramolecular pair forces cancel
// exactly in both (Newton's third law), so they are kept out of sums they contribute nothing to.
// The caller must group_sync before S.geno, the positions or own[] are touched again (part 0 still reads them).
// PRE: the J fragment's sums are loaded at the top of the tile that updates them (hides the read-modify-write latency, holds six
// registers across the tile) instead of just before the update.  Which is faster is a matter of ptxas's register allocation
// per variant (measured: the 16-warp scoring kernel 6.88e8 with, 6.75e8 without; the 12-warp ADADELTA kernel 6.02e8 with,
// 6.09e8 without).
template <bool GRAD, int K, int GOUT = 1, bool TM = false, bool PRE = false>
__device__ __forceinline__ float lane_eval(const LaneL& L, const GridDev& G, const ParDev& P, const LaneS& S, float* grad, int gs,
                                           bool wr, float& e_inter, float& e_intra, bool& gfin) {
    const float tx = S.geno[0], ty = S.geno[32], tz = S.geno[64];
    float qw = S.geno[96], qx = S.geno[128], qy = S.geno[160], qz = S.geno[192];
    const float qn2 = qw * qw + qx * qx + qy * qy + qz * qz;
    const bool badq = !(qn2 >= 1e-24f);
    if (badq) { qw = 1.f; qx = qy = qz = 0.f; }
    const float qi = badq ? 1.f : 1.0f / sqrtf(qn2);
    qw *= qi; qx *= qi; qy *= qi; qz *= qi;
    static_assert(!TM || K == 1, "tensor-memory positions are private to one warp");

    // (a1) pose: per-fragment transform = parent's o rotation about the reference-frame axis; positions relative to t.
    // With K > 1 part 0 builds the whole pose and the others wait: the chain of fragment transforms is serial, and
    // repeating it in every part costs issue slots (the scarce resource), an idle warp costs none.
    if (K == 1 || S.part == 0) {
        float m00 = 1.f - 2.f * (qy * qy + qz * qz), m01 = 2.f * (qx * qy - qw * qz), m02 = 2.f * (qx * qz + qw * qy);
        float m10 = 2.f * (qx * qy + qw * qz), m11 = 1.f - 2.f * (qx * qx + qz * qz), m12 = 2.f * (qy * qz - qw * qx);
        float m20 = 2.f * (qx * qz - qw * qy), m21 = 2.f * (qy * qz + qw * qx), m22 = 1.f - 2.f * (qx * qx + qy * qy);
        float m03 = 0.f, m13 = 0.f, m23 = 0.f;
        for (int f = 0; f < L.nfrag; ++f) {
            const int4 fi = L.fragi[3 * f];             // parent, depth|kids<<16, abeg, aend
            const int depth = fi.y & 0xffff;
            if (f > 0) {
                const int4 fa = L.fragi[3 * f + 1], fb = L.fragi[3 * f + 2];
                const float p0x = __int_as_float(fa.x), p0y = __int_as_float(fa.y), p0z = __int_as_float(fa.z);
                const float ux = __int_as_float(fb.x), uy = __int_as_float(fb.y), uz = __int_as_float(fb.z);
                const float4* st = S.oA + (depth - 1) * 3 * 32;
                const float4 r0 = st[0], r1 = st[32], r2 = st[64];
                const float b00 = r0.x, b01 = r0.y, b02 = r0.z, b03 = r0.w;
                const float b10 = r1.x, b11 = r1.y, b12 = r1.z, b13 = r1.w;
                const float b20 = r2.x, b21 = r2.y, b22 = r2.z, b23 = r2.w;
                float s, c;
                sincosf(S.geno[(7 + fa.w) * 32], &s, &c);
                const float k = 1.f - c;
                const float a00 = fmaf(k * ux, ux, c), a01 = fmaf(k * ux, uy, -s * uz), a02 = fmaf(k * ux, uz, s * uy);
                const float a10 = fmaf(k * ux, uy, s * uz), a11 = fmaf(k * uy, uy, c), a12 = fmaf(k * uy, uz, -s * ux);
                const float a20 = fmaf(k * ux, uz, -s * uy), a21 = fmaf(k * uy, uz, s * ux), a22 = fmaf(k * uz, uz, c);
                // x = B (A (y - p0) + p0) + b3  =>  M = B A,  m3 = B (p0 - A p0) + b3
                const float wx = p0x - (a00 * p0x + a01 * p0y + a02 * p0z), wy = p0y - (a10 * p0x + a11 * p0y + a12 * p0z),
                            wz = p0z - (a20 * p0x + a21 * p0y + a22 * p0z);
                m00 = b00 * a00 + b01 * a10 + b02 * a20; m01 = b00 * a01 + b01 * a11 + b02 * a21; m02 = b00 * a02 + b01 * a12 + b02 * a22;
                m10 = b10 * a00 + b11 * a10 + b12 * a20; m11 = b10 * a01 + b11 * a11 + b12 * a21; m12 = b10 * a02 + b11 * a12 + b12 * a22;
                m20 = b20 * a00 + b21 * a10 + b22 * a20; m21 = b20 * a01 + b21 * a11 + b22 * a21; m22 = b20 * a02 + b21 * a12 + b22 * a22;
                m03 = b00 * wx + b01 * wy + b02 * wz + b03;
                m13 = b10 * wx + b11 * wy + b12 * wz + b13;
                m23 = b20 * wx + b21 * wy + b22 * wz + b23;
            }
            if (fi.y >> 16) {                           // has children: push
                float4* st = S.oA + depth * 3 * 32;
                st[0] = make_float4(m00, m01, m02, m03);
                st[32] = make_float4(m10, m11, m12, m13);
                st[64] = make_float4(m20, m21, m22, m23);
            }
            for (int i = fi.z; i < fi.w; ++i) {
                const float4 a = L.atoms[i];
                pos_put<TM>(S, i, fmaf(m00, a.x, fmaf(m01, a.y, fmaf(m02, a.z, m03))), fmaf(m10, a.x, fmaf(m11, a.y, fmaf(m12, a.z, m13))),
                            fmaf(m20, a.x, fmaf(m21, a.y, fmaf(m22, a.z, m23))));
            }
        }
        for (int i = L.N; i < L.Npad; ++i) pos_put<TM>(S, i, 0.f, 0.f, 0.f);      // pad atoms: finite, in no pair
        if (TM) tm_wait_st();
    }

    group_sync<K>(S);                                   // the positions are in place
    // (a2) grid term, kLaneBI = 4 atoms per step: the 16 sector loads of a step are issued back to back before the first
    // is consumed (the lookups are pure L2 latency: one dependent round per step instead of one per atom); the
    // gradient goes straight into the (force, torque about t) sums of the atom's fragment, which initialises own[]
    float eg = 0.f;
    float RFx = 0, RFy = 0, RFz = 0, RTx = 0, RTy = 0, RTz = 0;     // grid force / torque about t over ALL atoms of this part
    const float ucx = (tx - G.ox) * G.inv_h, ucy = (ty - G.oy) * G.inv_h, ucz = (tz - G.oz) * G.inv_h;  // t in grid units
    {
        if (GRAD && K > 1)
            for (int f = 0; f < L.nfrag; ++f) { S.oA[f * 32] = make_float4(0.f, 0.f, 0.f, 0.f); S.oB[f * 32] = make_float2(0.f, 0.f); }
        float Fx = 0, Fy = 0, Fz = 0, Tx = 0, Ty = 0, Tz = 0;
        int cur = 0;
        for (int m = 2 * S.part; m < L.Npad / 2; m += 2 * K) {
            int tt[4];
            float q[4], rx[4], ry[4], rz[4];
            GridCell gc[4];
            F8 c[4][2];
            {
                const int4 t4 = *reinterpret_cast<const int4*>(L.types + 2 * m);      // cell set | frag << 8 ; -1 = pad
                tt[0] = t4.x; tt[1] = t4.y; tt[2] = t4.z; tt[3] = t4.w;
                Pos6 pa, pb;
                pos_issue<TM>(S, m, pa);
                pos_issue<TM>(S, m + 1, pb);
                pos_wait<TM>(pa, pb);
                rx[0] = pa.x0; rx[1] = pa.x1; rx[2] = pb.x0; rx[3] = pb.x1;
                ry[0] = pa.y0; ry[1] = pa.y1; ry[2] = pb.y0; ry[3] = pb.y1;
                rz[0] = pa.z0; rz[1] = pa.z1; rz[2] = pb.z0; rz[3] = pb.z1;
            }
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                q[a] = L.atoms[2 * m + a].w;
                gc[a] = grid_cell_u(G, tt[a] < 0 ? 0 : (tt[a] & 0xff), fmaf(rx[a], G.inv_h, ucx), fmaf(ry[a], G.inv_h, ucy), fmaf(rz[a], G.inv_h, ucz));
            }
#pragma unroll
            for (int a = 0; a < 4; ++a) grid_fetch(G, gc[a], c[a]);
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                float gx, gy, gz;
                const float e = grid_finish<GRAD>(G, P, gc[a], c[a], q[a], gx, gy, gz);
                if (tt[a] < 0) continue;                    // pad atom (warp-uniform): looked up, not counted
                eg += e;
                if (GRAD) {
                    const int f = tt[a] >> 8;
                    if (f != cur) {
                        own_flush<K>(S, cur, Fx, Fy, Fz, Tx, Ty, Tz);
                        RFx += Fx; RFy += Fy; RFz += Fz; RTx += Tx; RTy += Ty; RTz += Tz;
                        Fx = Fy = Fz = Tx = Ty = Tz = 0.f; cur = f;
                    }
                    Fx += gx; Fy += gy; Fz += gz;
                    Tx += ry[a] * gz - rz[a] * gy; Ty += rz[a] * gx - rx[a] * gz; Tz += rx[a] * gy - ry[a] * gx;
                }
            }
        }
        if (GRAD) {
            own_flush<K>(S, cur, Fx, Fy, Fz, Tx, Ty, Tz);
            RFx += Fx; RFy += Fy; RFz += Fz; RTx += Tx; RTy += Ty; RTz += Tz;
        }
    }

    // (a3) intramolecular pairs: register tiles; this warp's parts of the tile sequence.  The record of tile t+1 is
    // loaded while tile t computes (the tile array ends with a sentinel), and the J fragment's (force, torque) sums are
    // loaded at the top of the tile that updates them, so the read-modify-write of own[] is not waited for.
    f2 e2 = bc(0.f);
    for (int part = S.part; part < kLaneParts; part += K) {
        const PairK PK = make_pairk(P);
        const float4* rowp = L.rows + 2 * L.part_row[part];
        const f2 zero = bc(0.f);
        for (int kb = L.part_blk[part]; kb < L.part_blk[part + 1]; ++kb) {
            const int4 blk = L.blocks[2 * kb], bf = L.blocks[2 * kb + 1];   // b, tile_begin, tile_end, - ; frags of rows 0-3, 4-7
            uint2 tw = L.tiles[blk.y];
            float xi[kLaneBI], yi[kLaneBI], zi[kLaneBI];
            {
                Pos6 pi[kLaneBI / 2];
#pragma unroll
                for (int h2 = 0; h2 < kLaneBI / 2; ++h2) pos_issue<TM>(S, (kLaneBI / 2) * blk.x + h2, pi[h2]);
#pragma unroll
                for (int h2 = 0; h2 < kLaneBI / 2; h2 += 2) pos_wait<TM>(pi[h2], pi[h2 + 1]);
#pragma unroll
                for (int h2 = 0; h2 < kLaneBI / 2; ++h2) {
                    xi[2 * h2] = pi[h2].x0; xi[2 * h2 + 1] = pi[h2].x1; yi[2 * h2] = pi[h2].y0; yi[2 * h2 + 1] = pi[h2].y1;
                    zi[2 * h2] = pi[h2].z0; zi[2 * h2 + 1] = pi[h2].z1;
                }
            }
            f2 gix[kLaneBI], giy[kLaneBI], giz[kLaneBI];
#pragma unroll
            for (int r = 0; r < kLaneBI; ++r) gix[r] = giy[r] = giz[r] = zero;
            for (int t = blk.y; t < blk.z; ++t) {
                const uint2 cw = tw;
                tw = L.tiles[t + 1];                    // next tile (or the sentinel)
                Pos6 pj;
                pos_issue<TM>(S, cw.x & 0xff, pj);
                const int f0 = (cw.y >> 16) & 0xff, f1 = cw.y >> 24;
                float4 va = make_float4(0.f, 0.f, 0.f, 0.f);
                float2 vb = make_float2(0.f, 0.f);
                if (GRAD && PRE) { va = S.oA[f0 * 32]; vb = S.oB[f0 * 32]; }
                pos_wait<TM>(pj);
                const f2 xj = pk(pj.x0, pj.x1), yj = pk(pj.y0, pj.y1), zj = pk(pj.z0, pj.z1);
                f2 gjx = zero, gjy = zero, gjz = zero;
#pragma unroll
                for (int hf = 0; hf < kLaneBI / 2; ++hf) {   // a half = two rows = two independent chains in one basic block
                    if (cw.x & (0x100u << hf)) {
                        const float4 ra0 = rowp[0], rb0 = rowp[1], ra1 = rowp[2], rb1 = rowp[3];
                        rowp += 4;
                        const int r0 = 2 * hf, r1 = 2 * hf + 1;
                        if (!(cw.x & (0x1000u << hf))) {
                            pair_row<GRAD, false>(PK, bc(xi[r0]), bc(yi[r0]), bc(zi[r0]), xj, yj, zj, ra0, rb0, 0u, e2,
                                                  gix[r0], giy[r0], giz[r0], gjx, gjy, gjz);
                            pair_row<GRAD, false>(PK, bc(xi[r1]), bc(yi[r1]), bc(zi[r1]), xj, yj, zj, ra1, rb1, 0u, e2,
                                                  gix[r1], giy[r1], giz[r1], gjx, gjy, gjz);
                        } else {
                            pair_row<GRAD, true>(PK, bc(xi[r0]), bc(yi[r0]), bc(zi[r0]), xj, yj, zj, ra0, rb0, (cw.y >> (2 * r0)) & 3u,
                                                 e2, gix[r0], giy[r0], giz[r0], gjx, gjy, gjz);
                            pair_row<GRAD, true>(PK, bc(xi[r1]), bc(yi[r1]), bc(zi[r1]), xj, yj, zj, ra1, rb1, (cw.y >> (2 * r1)) & 3u,
                                                 e2, gix[r1], giy[r1], giz[r1], gjx, gjy, gjz);
                        }
                    }
                }
                if (GRAD) {                             // J side: gradients (a | b) of atoms (j0 | j1) -> fragment sums, the torque
                    float ax, bx, ay, by, az, bz;        // about t as chains of scalar fma on top of the loaded sums
                    unpk(gjx, ax, bx); unpk(gjy, ay, by); unpk(gjz, az, bz);
                    if (!PRE) { va = S.oA[f0 * 32]; vb = S.oB[f0 * 32]; }
                    const float t0x = fmaf(pj.y0, az, -pj.z0 * ay), t0y = fmaf(pj.z0, ax, -pj.x0 * az), t0z = fmaf(pj.x0, ay, -pj.y0 * ax);
                    if (f0 == f1) {
                        S.oA[f0 * 32] = make_float4((va.x + ax) + bx, (va.y + ay) + by, (va.z + az) + bz,
                                                    fmaf(pj.y1, bz, fmaf(-pj.z1, by, va.w + t0x)));
                        S.oB[f0 * 32] = make_float2(fmaf(pj.z1, bx, fmaf(-pj.x1, bz, vb.x + t0y)), fmaf(pj.x1, by, fmaf(-pj.y1, bx, vb.y + t0z)));
                    } else {                            // the J-pair straddles two fragments
                        S.oA[f0 * 32] = make_float4(va.x + ax, va.y + ay, va.z + az, va.w + t0x);
                        S.oB[f0 * 32] = make_float2(vb.x + t0y, vb.y + t0z);
                        own_add(S, f1, bx, by, bz, fmaf(pj.y1, bz, -pj.z1 * by), fmaf(pj.z1, bx, -pj.x1 * bz), fmaf(pj.x1, by, -pj.y1 * bx));
                    }
                }
            }
            if (GRAD) {                                 // I side: gi holds MINUS the gradient
                float Fx = 0, Fy = 0, Fz = 0, Tx = 0, Ty = 0, Tz = 0;
                auto frag_of_row = [&](int r) { return (int)(((r < 4 ? bf.x : bf.y) >> (8 * (r & 3))) & 0xff); };
#pragma unroll
                for (int r = 0; r < kLaneBI; ++r) {
                    const float gx = -hsum(gix[r]), gy = -hsum(giy[r]), gz = -hsum(giz[r]);
                    Fx += gx; Fy += gy; Fz += gz;
                    Tx += yi[r] * gz - zi[r] * gy; Ty += zi[r] * gx - xi[r] * gz; Tz += xi[r] * gy - yi[r] * gx;
                    const int fr = frag_of_row(r);
                    if (r == kLaneBI - 1 || fr != frag_of_row(r + 1)) {
                        own_add(S, fr, Fx, Fy, Fz, Tx, Ty, Tz);
                        Fx = Fy = Fz = Tx = Ty = Tz = 0.f;
                    }
                }
            }
        }
    }
    e_inter = eg;
    e_intra = hsum(e2);
    if (K > 1) {                                        // hand the partial sums to part 0
        float* ex = S.ex + 8 * S.part * 32;
        ex[0] = e_inter; ex[32] = e_intra;
        if (GRAD) { ex[64] = RFx; ex[96] = RFy; ex[128] = RFz; ex[160] = RTx; ex[192] = RTy; ex[224] = RTz; }
        group_sync<K>(S);
        if (S.part != 0) { gfin = true; return 0.f; }
        e_inter = 0.f; e_intra = 0.f;
        for (int k = 0; k < K; ++k) { e_inter += S.ex[(8 * k) * 32]; e_intra += S.ex[(8 * k + 1) * 32]; }
        if (GRAD) {
            RFx = RFy = RFz = RTx = RTy = RTz = 0.f;
            for (int k = 0; k < K; ++k) {
                const float* e8 = S.ex + 8 * k * 32;
                RFx += e8[64]; RFy += e8[96]; RFz += e8[128]; RTx += e8[160]; RTy += e8[192]; RTz += e8[224];
            }
            for (int f = 1; f < L.nfrag; ++f) {         // the root's own sums are not needed (grid totals above)
                float4 a = S.oA[f * 32];                // this is part 0
                float2 b = S.oB[f * 32];
                for (int k = 1; k < K; ++k) {
                    const float4 c = *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(S.oA + f * 32) + k * S.part_stride);
                    const float2 d = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(S.oB + f * 32) + k * S.part_stride);
                    a.x += c.x; a.y += c.y; a.z += c.z; a.w += c.w; b.x += d.x; b.y += d.y;
                }
                S.oA[f * 32] = a; S.oB[f * 32] = b;
            }
        }
    }
    float e = e_inter + e_intra;
    const float qnan = __int_as_float(0x7fc00000);
    if (badq) { e = qnan; e_inter = qnan; e_intra = qnan; }

    // (a4) back-propagation: subtree sums in place (children before parents), projection on the posed axes
    if (GRAD) {
        bool fin = true;
        for (int f = L.nfrag - 1; f > 0; --f) {
            const int4 fi = L.fragi[3 * f];
            const int tor = L.fragi[3 * f + 1].w, ab = L.fragi[3 * f + 2].w;
            const float4 oa = S.oA[f * 32];
            const float2 ob = S.oB[f * 32];
            const float Fx = oa.x, Fy = oa.y, Fz = oa.z, Tx = oa.w, Ty = ob.x, Tz = ob.y;
            const int ia = ab & 0xffff, ib = ab >> 16;
            float ax, ay, az, ux, uy, uz;
            pos_issue1<TM>(S, ia, ax, ay, az);
            pos_issue1<TM>(S, ib, ux, uy, uz);
            if (TM) tm_wait_ld(ax, ay, az, ux, uy, uz);
            ux -= ax; uy -= ay; uz -= az;
            const float un = rsqrtf(ux * ux + uy * uy + uz * uz);
            ux *= un; uy *= un; uz *= un;
            // torque about the pivot atom a: T - a x F
            const float px = Tx - (ay * Fz - az * Fy), py = Ty - (az * Fx - ax * Fz), pz = Tz - (ax * Fy - ay * Fx);
            float dt = ux * px + uy * py + uz * pz;
            if (badq) dt = qnan;
            fin = fin && isfinite(dt);
            if (GOUT == 1) { if (wr) grad[(6 + tor) * gs] = dt; }
            else reinterpret_cast<float*>(S.oA + f * 32)[0] = dt;     // fragment f's sums are consumed: its first slot carries dE/dtau
            if (fi.x != 0) own_add(S, fi.x, Fx, Fy, Fz, Tx, Ty, Tz);     // the root takes the grid totals instead
        }
        float g[6] = {RFx, RFy, RFz, RTx, RTy, RTz};
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            if (badq) g[d] = qnan;
            fin = fin && isfinite(g[d]);
            if (GOUT == 1) { if (wr) grad[d * gs] = g[d]; }
        }
        if (GOUT != 1) { S.oA[0] = make_float4(g[0], g[1], g[2], g[3]); S.oB[0] = make_float2(g[4], g[5]); }
        gfin = fin;
    }
    return e;
}

// ---------------------------------------------------------------- ADADELTA chain of this thread (R7)
struct LaneLS {             // global scratch columns of this thread: element d at [d*stride]
    float* best;            // [7+R]
    float* Eg2;             // [6+R]
    float* Ed2;             // [6+R]
    int stride;
};

// one component of the update (R7): accumulators in place, returns the step.  sqrt(a)/sqrt(b) as a*rsqrt(a)*rsqrt(b)
// with the MUFU forms (a, b >= ad_eps > 0): 3 instructions instead of two IEEE square roots and a division.
__device__ __forceinline__ float adadelta_component(const ParDev& P, float g, float& eg2, float& ed2) {
    eg2 = P.ad_rho * eg2 + (1.f - P.ad_rho) * g * g;
    const float a = ed2 + P.ad_eps;
    const float dl = -(a * frsqrt(a) * frsqrt(eg2 + P.ad_eps)) * g;
    ed2 = P.ad_rho * ed2 + (1.f - P.ad_rho) * dl * dl;
    return dl;
}

// Start genotype in S.geno (visible to the whole group).  Called by all K warps of the group; part 0 owns the chain's
// state (ls, in global scratch columns) and on return ls.best holds the best genotype seen; part 0 returns its energy
// (e_start if no finite evaluation happened) and the evaluations done.  `active` lanes run the chain; the others only
// keep the warp's control flow uniform.  The gradient never leaves shared memory (lane_eval, GOUT = 2).
template <int K, bool TM = false>
__device__ inline float lane_adadelta(const LaneL& L, const GridDev& G, const ParDev& P, const LaneS& S, const LaneLS& ls,
                                      bool active, float e_start, int& iters, float* trace, int trace_stride) {
    const int R = L.R, D = 6 + R, Gn = 7 + R;
    const bool lead = S.part == 0;
    float bestE = __int_as_float(0x7f800000);
    if (lead) {
        for (int d = 0; d < Gn; ++d) ls.best[d * ls.stride] = S.geno[d * 32];
        for (int d = 0; d < D; ++d) { ls.Eg2[d * ls.stride] = 0.f; ls.Ed2[d * ls.stride] = 0.f; }
    }
    bool live = active;
    int it = 0;
    iters = 0;
    for (; it < P.lsit; ++it) {
        if (!__any_sync(kFull, live)) break;            // same decision in every warp of the group
        float ei, ea;
        bool gfin = true;
        const float e = lane_eval<true, K, 2, TM>(L, G, P, S, nullptr, 0, false, ei, ea, gfin);
        if (lead) {
            if (live) {
                if (trace) trace[it * trace_stride] = e;
                ++iters;
                if (!(isfinite(e) && gfin)) live = false;
            }
            if (live) {
                if (e < bestE) {
                    bestE = e;
                    for (int d = 0; d < Gn; ++d) ls.best[d * ls.stride] = S.geno[d * 32];
                }
                // the accumulator columns live in global memory (L2): a chunk of 8 components is loaded before the
                // first store, so the chunk costs one round trip instead of one per component
                float w[3];
                {                                       // rigid-body block: d = 0..5, gradient in oA[0], oB[0]
                    const float4 ga = S.oA[0];
                    const float2 gb = S.oB[0];
                    const float gr[6] = {ga.x, ga.y, ga.z, ga.w, gb.x, gb.y};
                    float av[6], bv[6];
#pragma unroll
                    for (int d = 0; d < 6; ++d) { av[d] = ls.Eg2[d * ls.stride]; bv[d] = ls.Ed2[d * ls.stride]; }
#pragma unroll
                    for (int d = 0; d < 6; ++d) {
                        const float dl = adadelta_component(P, gr[d], av[d], bv[d]);
                        ls.Eg2[d * ls.stride] = av[d]; ls.Ed2[d * ls.stride] = bv[d];
                        if (d < 3) S.geno[d * 32] += dl; else w[d - 3] = dl;
                    }
                }
                if (TM) {                                   // chain state in shared memory: no round trips to batch
                    for (int f = 1; f < L.nfrag; ++f) {
                        const int d = 6 + L.fragi[3 * f + 1].w;
                        float av = ls.Eg2[d * 32], bv = ls.Ed2[d * 32];
                        const float dl = adadelta_component(P, reinterpret_cast<const float*>(S.oA + f * 32)[0], av, bv);
                        ls.Eg2[d * 32] = av; ls.Ed2[d * 32] = bv;
                        float* t = S.geno + (d + 1) * 32;
                        *t = wrap_pi(*t + dl);
                    }
                } else
                for (int f0 = 1; f0 < L.nfrag; f0 += 8) {  // torsions: fragment f's torsion gradient in oA[f*32].x
                    float av[8], bv[8];
                    int dd[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int f = min(f0 + k, L.nfrag - 1);
                        dd[k] = 6 + L.fragi[3 * f + 1].w;
                        av[k] = ls.Eg2[dd[k] * ls.stride]; bv[k] = ls.Ed2[dd[k] * ls.stride];
                    }
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int f = f0 + k;
                        if (f < L.nfrag) {
                            const float dl = adadelta_component(P, reinterpret_cast<const float*>(S.oA + f * 32)[0], av[k], bv[k]);
                            ls.Eg2[dd[k] * ls.stride] = av[k]; ls.Ed2[dd[k] * ls.stride] = bv[k];
                            float* t = S.geno + (dd[k] + 1) * 32;
                            *t = wrap_pi(*t + dl);
                        }
                    }
                }
                const float th = sqrtf(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
                float sh, ch;
                sincosf(0.5f * th, &sh, &ch);
                const float k = th > 1e-12f ? sh / th : 0.5f;
                const float q[4] = {S.geno[96], S.geno[128], S.geno[160], S.geno[192]};
                float nq[4];
                rotate_quat(ch, k * w[0], k * w[1], k * w[2], q, nq);
                S.geno[96] = nq[0]; S.geno[128] = nq[1]; S.geno[160] = nq[2]; S.geno[192] = nq[3];
            }
            if (K > 1) S.ex[(8 * K) * 32] = live ? 1.f : 0.f;
        }
        group_sync<K>(S);                               // new genotype and live flag visible; part 0 is done with own[]
        if (K > 1) live = S.ex[(8 * K) * 32] != 0.f;
    }
    return isfinite(bestE) ? bestE : e_start;
}

// ---------------------------------------------------------------- Solis-Wets chain of this thread (R11)
// Start genotype in S.geno (visible to the whole group) with carried energy e_start.  Every pass of the loop is ONE
// evaluation of the whole warp; each lane runs its own state machine (phase 0: try x (+) delta, phase 1: try x (-) delta),
// so a lane whose first trial succeeded draws its next step at once instead of idling through the other lanes'
// second trial.  Part 0 owns the state: x in ls.best, bias in ls.Eg2, delta in ls.Ed2 (global scratch columns).
// On return ls.best holds the accepted genotype; part 0 returns its energy and the evaluations done.
template <int K, bool TM = false>
__device__ inline float lane_solis_wets(const LaneL& L, const GridDev& G, const ParDev& P, const LaneS& S, const LaneLS& ls,
                                        bool active, float e_start, unsigned long long seed, uint32_t id, uint32_t gen, int& evals,
                                        float* trace, int trace_stride) {
    const int R = L.R, D = 6 + R, Gn = 7 + R, nq = (D + 3) / 4;
    const bool lead = S.part == 0;
    float E = e_start, rho = P.sw_rho0;
    int ns = 0, nf = 0, it = 0, phase = 0;
    evals = 0;
    if (lead) {
        for (int d = 0; d < Gn; ++d) ls.best[d * ls.stride] = S.geno[d * 32];
        for (int d = 0; d < D; ++d) ls.Eg2[d * ls.stride] = 0.f;
    }
    bool live = active && P.lsit > 0 && !(rho < P.sw_rho_lb);
    for (;;) {
        float sg = 1.f;
        if (lead && live) {                             // candidate = x (+) sg*delta into S.geno
            if (phase == 0) {
                for (int q = 0; q < nq; ++q) {
                    const uint4 r = draw4(seed, (uint32_t)(it * nq + q), kSolisWets, id, gen);
                    for (int w = 0; w < 4 && 4 * q + w < D; ++w) {
                        const int d = 4 * q + w;
                        const float xi = 2.f * u01(pick_word(r, w)) - 1.f;
                        ls.Ed2[d * ls.stride] = rho * (d < 3 ? P.dmov : P.dang) * xi + ls.Eg2[d * ls.stride];
                    }
                }
            } else {
                sg = -1.f;
            }
            for (int d = 0; d < 3; ++d) S.geno[d * 32] = ls.best[d * ls.stride] + sg * ls.Ed2[d * ls.stride];
            const float wx = sg * ls.Ed2[3 * ls.stride], wy = sg * ls.Ed2[4 * ls.stride], wz = sg * ls.Ed2[5 * ls.stride];
            const float th = sqrtf(wx * wx + wy * wy + wz * wz);
            float sh, ch;
            sincosf(0.5f * th, &sh, &ch);
            const float k = th > 1e-12f ? sh / th : 0.5f;
            const float q0[4] = {ls.best[3 * ls.stride], ls.best[4 * ls.stride], ls.best[5 * ls.stride], ls.best[6 * ls.stride]};
            float nq4[4];
            rotate_quat(ch, k * wx, k * wy, k * wz, q0, nq4);
            S.geno[96] = nq4[0]; S.geno[128] = nq4[1]; S.geno[160] = nq4[2]; S.geno[192] = nq4[3];
            for (int d = 6; d < D; ++d) S.geno[(d + 1) * 32] = wrap_pi(ls.best[(d + 1) * ls.stride] + sg * ls.Ed2[d * ls.stride]);
        }
        if (K > 1 && lead) S.ex[(8 * K) * 32] = live ? 1.f : 0.f;
        group_sync<K>(S);                               // candidate and live flag visible; part 0 is done with the last pass
        if (K > 1) live = S.ex[(8 * K) * 32] != 0.f;
        if (!__any_sync(kFull, live)) break;            // same decision in every warp of the group
        float ei, ea;
        bool gfin = true;
        const float e = lane_eval<false, K, 1, TM>(L, G, P, S, nullptr, 1, false, ei, ea, gfin);
        if (lead && live) {
            ++evals;
            const bool ok = e < E;
            bool done = true;
            if (ok) {
                E = e;
                for (int d = 0; d < Gn; ++d) ls.best[d * ls.stride] = S.geno[d * 32];
                for (int d = 0; d < D; ++d)
                    ls.Eg2[d * ls.stride] = P.sw_bias_keep * ls.Eg2[d * ls.stride] + P.sw_bias_gain * (sg * ls.Ed2[d * ls.stride]);
                ++ns; nf = 0;
            } else if (phase == 0) {
                phase = 1; done = false;
            } else {
                for (int d = 0; d < D; ++d) ls.Eg2[d * ls.stride] *= P.sw_bias_decay;
                ++nf; ns = 0;
            }
            if (done) {
                phase = 0;
                if (ns >= P.sw_max_succ) { rho *= P.sw_expand; ns = 0; }
                else if (nf >= P.sw_max_fail) { rho *= P.sw_contract; nf = 0; }
                if (trace) trace[it * trace_stride] = E;
                ++it;
                live = it < P.lsit && !(rho < P.sw_rho_lb);
            }
        }
    }
    return E;
}

}  // namespace adock
