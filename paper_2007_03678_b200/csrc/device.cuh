// device.cuh -- sm_100a device code of the hot path: pose builder, grid interpolator, intramolecular
// pair evaluator, reductions and gradient back-propagation (R3-R6), ADADELTA (R7),
// Philox4x32-10 (R8) and the GA operators (R9).  One WARP per individual; the ligand image (topology.hpp)
// is staged once per CTA into shared memory by a bulk async copy (TMA, UBLKCP) and shared by its warps.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "topology.hpp"

namespace adock {

constexpr unsigned kFull = 0xffffffffu;
constexpr float kPi = 3.14159265358979323846f;
constexpr float kTwoPi = 6.28318530717958647692f;

struct GridDev {
    const float4* cells;    // [2T][nz][ny-1][nx-1] xy-patch cells of one 32-byte sector (2 float4): the pair (a_t, pm) at the
                            // nodes (ix,iy), (ix+1,iy), (ix,iy+1), (ix+1,iy+1) of plane iz, for cell set 2t + s;
                            // pm = elec + desolv (s = 0: atoms with q >= 0) or elec - desolv (s = 1: q < 0)
    long long set_stride;   // float4 units between cell sets
    int nx, ny, nz, T;
    float inv_h, h;
    float ox, oy, oz;
    float bx, by, bz;       // box extents h*(n-1)
};

struct ParDev {             // adock_params with the per-pair constants folded
    float elec_sqrt, diel_A, diel_B, diel_k, BlamB, mlamB_log2e;   // elec_sqrt = sqrt(elec_scale); BlamB = B*lambda*B
    float log2_dk;          // log2(diel_k): the lane kernels fold k into the exponent of k exp(-lambda B r)
    float diel_As, diel_Bs; // lane kernels: A/s, B/s with s = B*lambda*B, so that 1/(den*(A/s*den + B/s)) = s/(den num) carries
                            // the factor of d(eps)/dr; the row coefficients qq of the lane image are divided by s (lane_elec_fold)
    float inv_sig2, mhalf_inv_sig2_log2e;
    float rmin2, k_wall, k_wall_h;
    float ad_rho, ad_eps;
    float tourn_prob, xover_rate, mut_rate, dmov, dang;
    int lsit;
    // R11 Solis-Wets, R12 autostop
    int ls_method, sw_max_succ, sw_max_fail, autostop, as_window;
    float sw_rho0, sw_rho_lb, sw_expand, sw_contract, sw_bias_keep, sw_bias_gain, sw_bias_decay, as_tol;
};
constexpr int kAsMaxWindow = 64;

// ---------------------------------------------------------------- shared-memory views
struct LigS {
    const float4* atoms;    // (x0 - pivot, q) by position
    const uint32_t* meta;   // type | frag<<8 ; 0xffffffff = hole
    const uint16_t* fragatoms;  // positions grouped by fragment
    const float4* fg;       // FragGeom as 2 float4
    const int4* fi;         // FragIdx
    const uint4* pairs;     // PairRec rounds
    int N, R, nfrag, nrounds, npos, nfull, systolic;
};

struct WarpS {
    float* geno;            // [Gpad]
    float* grad;            // [Dpad]  (also the ADADELTA step)
    float* best;            // [Gpad]
    float2* sc;             // [nfrag] sin,cos of the fragment's torsion
    float4* fragT;          // [nfrag][3] rows of the 3x4 fragment transform
    float4* fragAx;         // [nfrag][2] posed axis, posed pivot point - t
    float4* fragFT;         // [nfrag][2] force, torque about the fragment's own pivot point
    float* blk;             // pose block, 256 floats per 32 atoms: x|y|z|q|gx|gy|gz|-  (32 each), so atom a
                            // lives at slot(a) = (a>>5)*256 + (a&31) and distinct a mod 32 hit distinct banks
};
constexpr int kX = 0, kY = 32, kZ = 64, kQ = 96, kGX = 128, kGY = 160, kGZ = 192;
__host__ __device__ inline int atom_slot_dev(int a) { return (a >> 5) * 256 + (a & 31); }

__host__ __device__ inline int pad4(int x) { return (x + 3) & ~3; }
// floats of per-warp scratch for a ligand with N atoms, nfrag fragments, R torsions
__host__ __device__ inline int warp_scratch_floats(int N, int nfrag, int R) {
    return 2 * pad4(7 + R) + pad4(6 + R) + pad4(2 * nfrag) + nfrag * 28 + ((N + 31) / 32) * 256;
}

__device__ inline LigS lig_view(const unsigned char* blob) {
    const LigHeader* h = reinterpret_cast<const LigHeader*>(blob);
    LigS L;
    L.atoms = reinterpret_cast<const float4*>(blob + h->off_atoms);
    L.meta = reinterpret_cast<const uint32_t*>(blob + h->off_meta);
    L.fg = reinterpret_cast<const float4*>(blob + h->off_frag);
    L.fi = reinterpret_cast<const int4*>(blob + h->off_fragidx);
    L.pairs = reinterpret_cast<const uint4*>(blob + h->off_pairs);
    L.fragatoms = reinterpret_cast<const uint16_t*>(blob + h->off_fragatoms);
    L.N = h->N; L.R = h->R; L.nfrag = h->nfrag; L.nrounds = h->nrounds; L.npos = h->npos; L.nfull = h->nfull; L.systolic = h->systolic;
    return L;
}

__device__ inline WarpS warp_view(float* base, const LigS& L) {
    WarpS S;
    int Gp = pad4(7 + L.R), Dp = pad4(6 + L.R);
    S.geno = base; base += Gp;
    S.best = base; base += Gp;
    S.grad = base; base += Dp;
    S.sc = reinterpret_cast<float2*>(base); base += pad4(2 * L.nfrag);
    S.fragT = reinterpret_cast<float4*>(base); base += 12 * L.nfrag;
    S.fragAx = reinterpret_cast<float4*>(base); base += 8 * L.nfrag;
    S.fragFT = reinterpret_cast<float4*>(base); base += 8 * L.nfrag;
    S.blk = base;
    return S;
}

// ---------------------------------------------------------------- TMA bulk copy of the ligand image
__device__ inline uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// All threads of the CTA call this; returns after the image is visible in shared memory.
__device__ inline void stage_ligand(unsigned char* dst, const unsigned char* src, int bytes, uint64_t* bar, uint32_t phase) {
    if (threadIdx.x == 0) {
        if (phase == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bar)));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                     "l"(src), "r"(bytes), "r"(smem_u32(bar))
                     : "memory");
    }
    __syncthreads();
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(phase & 1u)
            : "memory");
    }
}

// Several images in one transaction: image s (src(s), bytes(s), both multiples of 16) lands at dst + s*slot_bytes.
// All threads of the CTA call this once (phase 0); returns after every image is visible in shared memory.
template <class SrcFn>
__device__ inline void stage_images(unsigned char* dst, int slot_bytes, int nimg, SrcFn src, uint64_t* bar) {
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        uint32_t total = 0;
        for (int s = 0; s < nimg; ++s) { const unsigned char* p; int b; src(s, p, b); total += (uint32_t)b; }
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(total) : "memory");
        for (int s = 0; s < nimg; ++s) {
            const unsigned char* p; int b;
            src(s, p, b);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                             smem_u32(dst + (size_t)s * slot_bytes)),
                         "l"(p), "r"(b), "r"(smem_u32(bar))
                         : "memory");
        }
    }
    __syncthreads();
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(0u)
            : "memory");
    }
}

// ---------------------------------------------------------------- packed f32x2 (FFMA2 / FMUL2 / FADD2)
struct f2 { unsigned long long v; };
__device__ __forceinline__ f2 pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f2 bc(float x) { return pk(x, x); }
__device__ __forceinline__ void unpk(f2 a, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { f2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return d; }
__device__ __forceinline__ f2 neg2(f2 a) { f2 d; d.v = a.v ^ 0x8000000080000000ull; return d; }
__device__ __forceinline__ float hsum(f2 a) { float l, h; unpk(a, l, h); return l + h; }
__device__ __forceinline__ f2 ld2(const float2* p) { const float2 v = *p; return pk(v.x, v.y); }

// ---------------------------------------------------------------- grid term (R4)
// One routine for every kernel family, in three stages so that a caller can issue the loads of several atoms before
// consuming any of them: grid_cell (clamp, cell index, fractions), grid_fetch (2 sector loads), grid_finish
// (trilinear value and gradient).
// The atom's energy is a_t + q*elec + |q|*desolv = a_t + q*(elec + sign(q)*desolv): the maps are re-laid-out once
// (relayout_kernel) into cell sets indexed by (type, sign of the charge) holding the pair (a_t, pm = elec +- desolv) per
// node, so the two fields an atom interpolates arrive as the two halves of packed f32x2 operands, register-aligned
// straight from the load: no per-corner mixing and no packing moves.  The small field pm (O(1..10)) and the affinity
// field (up to the 1e5 clamp) stay in separate halves until the very end, so the small one is never rounded to the
// ulp of the large one before the corner differences that make the gradient are taken.
// A cell is the 2x2 (x, y) patch of one z-plane = one aligned 32-byte sector, fetched whole by one LDG.256: a lookup is
// two sector loads (planes iz, iz+1), all 64 bytes used.  Measured (profiles/r02_grid_layout.md): the cost of the grid
// phase is per load request and lane (L1 miss handling), not per byte -- a 256-bit sector load is faster than a 128-bit
// load of half of it -- so the layout minimises requests; the price is every node stored four times per set.
// The lookups of a warp are scattered over the maps (32 lanes = 32 poses), so a line brought into L1 is not touched
// again before it is evicted: L1::no_allocate skips the allocation (profiles/r01b_grid_load_variants.md).
struct F8 { float4 lo, hi; };
__device__ __forceinline__ F8 ld_cell(const float4* p) {
    F8 r;
    asm("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(r.lo.x), "=f"(r.lo.y), "=f"(r.lo.z), "=f"(r.lo.w), "=f"(r.hi.x), "=f"(r.hi.y), "=f"(r.hi.z), "=f"(r.hi.w)
        : "l"(p));
    return r;
}
struct GridCell {
    const float4* base;     // cell (iz, iy, ix) of the atom's cell set
    float fx, fy, fz;       // fractions inside the cell
    float ox, oy, oz;       // signed distance outside the box in grid units (0 inside)
};
// `set` = 2*type + (q < 0)
// (ux, uy, uz) = position in grid units
__device__ __forceinline__ GridCell grid_cell_u(const GridDev& G, int set, float ux, float uy, float uz) {
    const float cx = fminf(fmaxf(ux, 0.f), (float)(G.nx - 1)), cy = fminf(fmaxf(uy, 0.f), (float)(G.ny - 1)),
                cz = fminf(fmaxf(uz, 0.f), (float)(G.nz - 1));
    const int ix = min((int)cx, G.nx - 2), iy = min((int)cy, G.ny - 2), iz = min((int)cz, G.nz - 2);
    GridCell c;
    c.fx = cx - (float)ix; c.fy = cy - (float)iy; c.fz = cz - (float)iz;
    c.ox = ux - cx; c.oy = uy - cy; c.oz = uz - cz;
    c.base = G.cells + (long long)set * G.set_stride + ((long long)(iz * (G.ny - 1) + iy) * (G.nx - 1) + ix) * 2;
    return c;
}
__device__ __forceinline__ GridCell grid_cell(const GridDev& G, int set, float x, float y, float z) {
    return grid_cell_u(G, set, (x - G.ox) * G.inv_h, (y - G.oy) * G.inv_h, (z - G.oz) * G.inv_h);
}
// v[0] = plane iz, v[1] = plane iz+1; each {a,pm}(ix,iy) {a,pm}(ix+1,iy) | {a,pm}(ix,iy+1) {a,pm}(ix+1,iy+1)
__device__ __forceinline__ void grid_fetch(const GridDev& G, const GridCell& c, F8 (&v)[2]) {
    v[0] = ld_cell(c.base);
    v[1] = ld_cell(c.base + (long long)(G.ny - 1) * (G.nx - 1) * 2);
}
// value and (GRAD) gradient in kcal/mol/A of the atom's grid energy; packed halves (affinity | pm), joined as
// lo + q*hi at the very end
template <bool GRAD>
__device__ __forceinline__ float grid_finish(const GridDev& G, const ParDev& P, const GridCell& c, const F8 (&v)[2], float q,
                                             float& gx, float& gy, float& gz) {
    const f2 a00 = pk(v[0].lo.x, v[0].lo.y), b00 = pk(v[0].lo.z, v[0].lo.w), a01 = pk(v[0].hi.x, v[0].hi.y), b01 = pk(v[0].hi.z, v[0].hi.w);
    const f2 a10 = pk(v[1].lo.x, v[1].lo.y), b10 = pk(v[1].lo.z, v[1].lo.w), a11 = pk(v[1].hi.x, v[1].hi.y), b11 = pk(v[1].hi.z, v[1].hi.w);
    const f2 fx = bc(c.fx), fy = bc(c.fy), fz = bc(c.fz);
    const f2 d00 = sub2(b00, a00), d01 = sub2(b01, a01), d10 = sub2(b10, a10), d11 = sub2(b11, a11);       // d/dfx per row
    const f2 v00 = fma2(fx, d00, a00), v01 = fma2(fx, d01, a01), v10 = fma2(fx, d10, a10), v11 = fma2(fx, d11, a11);
    const f2 e0 = sub2(v01, v00), e1 = sub2(v11, v10);                                                    // d/dfy per z-plane
    const f2 w0 = fma2(fy, e0, v00), w1 = fma2(fy, e1, v10);
    const f2 dz = sub2(w1, w0);
    float lo, hi;
    unpk(fma2(fz, dz, w0), lo, hi);
    float val = fmaf(q, hi, lo);
    val = fmaf(P.k_wall_h, fabsf(c.ox) + fabsf(c.oy) + fabsf(c.oz), val);
    if (GRAD) {
        const f2 dx0 = fma2(fy, sub2(d01, d00), d00), dx1 = fma2(fy, sub2(d11, d10), d10);
        unpk(fma2(fz, sub2(dx1, dx0), dx0), lo, hi);
        const float dfx = fmaf(q, hi, lo);
        unpk(fma2(fz, sub2(e1, e0), e0), lo, hi);
        const float dfy = fmaf(q, hi, lo);
        unpk(dz, lo, hi);
        const float dfz = fmaf(q, hi, lo);
        gx = (c.ox != 0.f) ? copysignf(P.k_wall, c.ox) : dfx * G.inv_h;
        gy = (c.oy != 0.f) ? copysignf(P.k_wall, c.oy) : dfy * G.inv_h;
        gz = (c.oz != 0.f) ? copysignf(P.k_wall, c.oz) : dfz * G.inv_h;
    }
    return val;
}
// the three stages for one atom
template <bool GRAD>
__device__ __forceinline__ float grid_atom(const GridDev& G, const ParDev& P, int set, float q, float x, float y, float z,
                                           float& gx, float& gy, float& gz) {
    const GridCell c = grid_cell(G, set, x, y, z);
    F8 v[2];
    grid_fetch(G, c, v);
    return grid_finish<GRAD>(G, P, c, v, q, gx, gy, gz);
}

// The team kernel looks an atom up after the pair rounds and asks for the two sectors before them (the cell is computed
// twice; nothing is held in registers over the pair loop): prefetch into L1, then loads that may hit there.
__device__ __forceinline__ void grid_prefetch(const GridDev& G, const GridCell& c) {
    asm volatile("prefetch.global.L1 [%0];" ::"l"(c.base));
    asm volatile("prefetch.global.L1 [%0];" ::"l"(c.base + (long long)(G.ny - 1) * (G.nx - 1) * 2));
}
__device__ __forceinline__ F8 ld_cell_l1(const float4* p) {
    F8 r;
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(r.lo.x), "=f"(r.lo.y), "=f"(r.lo.z), "=f"(r.lo.w), "=f"(r.hi.x), "=f"(r.hi.y), "=f"(r.hi.z), "=f"(r.hi.w)
        : "l"(p));
    return r;
}
template <bool GRAD>
__device__ __forceinline__ float grid_atom_l1(const GridDev& G, const ParDev& P, int set, float q, float x, float y, float z,
                                              float& gx, float& gy, float& gz) {
    const GridCell c = grid_cell(G, set, x, y, z);
    F8 v[2];
    v[0] = ld_cell_l1(c.base);
    v[1] = ld_cell_l1(c.base + (long long)(G.ny - 1) * (G.nx - 1) * 2);
    return grid_finish<GRAD>(G, P, c, v, q, gx, gy, gz);
}

// single-instruction MUFU forms (flush-to-zero): reciprocal, reciprocal square root, 2^x
__device__ __forceinline__ float frcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float frsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float fex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// eight sums at once: returns, in every lane, the sum over the warp of v[(lane >> 2) & 7] (9 shuffles; fixed order)
__device__ __forceinline__ float warp_sum8(const float (&v)[8], int lane) {
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
    float a[4], c[2];
#pragma unroll
    for (int k = 0; k < 4; ++k) a[k] = (b4 ? v[k + 4] : v[k]) + __shfl_xor_sync(kFull, b4 ? v[k] : v[k + 4], 16);
#pragma unroll
    for (int k = 0; k < 2; ++k) c[k] = (b3 ? a[k + 2] : a[k]) + __shfl_xor_sync(kFull, b3 ? a[k] : a[k + 2], 8);
    float d = (b2 ? c[1] : c[0]) + __shfl_xor_sync(kFull, b2 ? c[0] : c[1], 4);
    d += __shfl_xor_sync(kFull, d, 2);
    d += __shfl_xor_sync(kFull, d, 1);
    return d;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

// ---------------------------------------------------------------- intramolecular pair term (R5): one warp round
// Each lane evaluates one pair (i,j) of the round and adds +f to atom i, then -f to atom j.  Within a round no
// atom occurs twice on a side (topology.hpp), so the read-modify-writes need no atomics and their order is fixed.
// The arithmetic of a round (pair_compute) touches only positions and charges, so several rounds can be in flight at
// once; the force updates (pair_apply) then run round by round in the fixed order.
struct PairOut { int oi, oj; float fx, fy, fz, e; bool valid; };        // oi, oj: the atoms' offsets in S.blk
// the pair of record `rec` with atom i given by value (position, scaled charge) and atom j read from the pose block
template <bool GRAD, bool MAYPAD>
__device__ __forceinline__ PairOut pair_core(const ParDev& P, const uint4 rec, float xi, float yi, float zi, float qi, const float* blk) {
    const bool valid = !MAYPAD || ((rec.x >> 23) & 1u);
    const int oi = (int)(rec.x & 0x7ffu), oj = (int)((rec.x >> 11) & 0x7ffu);
    const float* pj = blk + oj;
    const float dx = xi - pj[kX], dy = yi - pj[kY], dz = zi - pj[kZ];
    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
    const float r2c = fmaxf(r2, P.rmin2);
    const float rinv = frsqrt(r2c);
    const float rr = r2c * rinv;
    const float rinv2 = rinv * rinv;
    const float r6 = rinv2 * rinv2 * rinv2, r12 = r6 * r6;
    const bool hb = (rec.x >> 22) & 1u;
    const float rA = hb ? r12 * r2c : r6;
    const float c12 = __uint_as_float(rec.y), cA = __uint_as_float(rec.z), ds = __uint_as_float(rec.w);
    const float u12 = c12 * r12, uA = cA * rA;
    const float ex = fex2(rr * P.mlamB_log2e);
    const float rden = frcp(fmaf(P.diel_k, ex, 1.f));
    const float eps = fmaf(P.diel_B, rden, P.diel_A);
    const float inv_er = rinv * frcp(eps);
    const float eel = qi * pj[kQ] * inv_er;                     // charges are stored pre-scaled by sqrt(elec_scale)
    const float egs = ds * fex2(r2c * P.mhalf_inv_sig2_log2e);
    const float e = (u12 - uA) + eel + egs;
    PairOut o;
    o.fx = o.fy = o.fz = 0.f;
    if (GRAD) {
        const float dv = fmaf(hb ? 10.f : 6.f, uA, -12.f * u12);            // r * d(vdw)/dr
        const float deps = P.BlamB * (1.f - rden) * rden;
        const float del = -eel * fmaf(deps, rr, eps) * inv_er;             // d(elec)/dr
        const float dds = -rr * P.inv_sig2 * egs;                          // d(desolv)/dr
        const float fs = (r2 >= P.rmin2) ? fmaf(dv, rinv, del + dds) * rinv : 0.f;
        o.fx = fs * dx; o.fy = fs * dy; o.fz = fs * dz;
    }
    o.oi = oi; o.oj = oj; o.valid = valid;
    o.e = valid ? e : 0.f;
    return o;
}
template <bool GRAD, bool MAYPAD>
__device__ __forceinline__ PairOut pair_compute(const LigS& L, const ParDev& P, const WarpS& S, int r, int lane) {
    const uint4 rec = L.pairs[r * 32 + lane];
    const float* pi = S.blk + (rec.x & 0x7ffu);
    return pair_core<GRAD, MAYPAD>(P, rec, pi[kX], pi[kY], pi[kZ], pi[kQ], S.blk);
}
// Two records of the same atom i (two partners ja, jb) as packed f32x2 arithmetic (lower half = ja): pair_core's
// expressions two at a time; MUFU, min / max and selects on the halves.
__device__ __forceinline__ void pair_core2(const ParDev& P, const uint4 reca, const uint4 recb, float xi, float yi, float zi, float qi,
                                           const float* blk, PairOut& oa, PairOut& ob) {
    oa.valid = (reca.x >> 23) & 1u; ob.valid = (recb.x >> 23) & 1u;
    oa.oj = (int)((reca.x >> 11) & 0x7ffu); ob.oj = (int)((recb.x >> 11) & 0x7ffu);
    const float* pja = blk + oa.oj, *pjb = blk + ob.oj;
    const f2 dx = sub2(bc(xi), pk(pja[kX], pjb[kX])), dy = sub2(bc(yi), pk(pja[kY], pjb[kY])), dz = sub2(bc(zi), pk(pja[kZ], pjb[kZ]));
    const f2 qq = mul2(bc(qi), pk(pja[kQ], pjb[kQ]));
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, mul2(dz, dz)));
    float r2a, r2b, ta, tb, sa, sb;
    unpk(r2, r2a, r2b);
    const float r2ca = fmaxf(r2a, P.rmin2), r2cb = fmaxf(r2b, P.rmin2);
    const f2 r2c = pk(r2ca, r2cb), rinv = pk(frsqrt(r2ca), frsqrt(r2cb));
    const f2 rr = mul2(r2c, rinv), rinv2 = mul2(rinv, rinv);
    const f2 r6 = mul2(mul2(rinv2, rinv2), rinv2), r12 = mul2(r6, r6);
    const bool hba = (reca.x >> 22) & 1u, hbb = (recb.x >> 22) & 1u;
    unpk(mul2(r12, r2c), ta, tb);
    unpk(r6, sa, sb);
    const f2 rA = pk(hba ? ta : sa, hbb ? tb : sb);
    const f2 u12 = mul2(pk(__uint_as_float(reca.y), __uint_as_float(recb.y)), r12), uA = mul2(pk(__uint_as_float(reca.z), __uint_as_float(recb.z)), rA);
    unpk(mul2(rr, bc(P.mlamB_log2e)), ta, tb);
    unpk(fma2(bc(P.diel_k), pk(fex2(ta), fex2(tb)), bc(1.f)), ta, tb);
    const f2 rden = pk(frcp(ta), frcp(tb));
    const f2 eps = fma2(bc(P.diel_B), rden, bc(P.diel_A));
    unpk(eps, ta, tb);
    const f2 inv_er = mul2(rinv, pk(frcp(ta), frcp(tb)));
    const f2 eel = mul2(qq, inv_er);
    unpk(mul2(r2c, bc(P.mhalf_inv_sig2_log2e)), ta, tb);
    const f2 egs = mul2(pk(__uint_as_float(reca.w), __uint_as_float(recb.w)), pk(fex2(ta), fex2(tb)));
    unpk(add2(add2(sub2(u12, uA), eel), egs), ta, tb);
    oa.e = oa.valid ? ta : 0.f; ob.e = ob.valid ? tb : 0.f;
    const f2 dv = fma2(pk(hba ? 10.f : 6.f, hbb ? 10.f : 6.f), uA, mul2(bc(-12.f), u12));       // r * d(vdw)/dr
    const f2 deps = mul2(mul2(bc(P.BlamB), sub2(bc(1.f), rden)), rden);
    const f2 del = mul2(mul2(neg2(eel), fma2(deps, rr, eps)), inv_er);                         // d(elec)/dr
    const f2 dds = mul2(mul2(neg2(rr), bc(P.inv_sig2)), egs);                                  // d(desolv)/dr
    unpk(mul2(fma2(dv, rinv, add2(del, dds)), rinv), ta, tb);
    const f2 fs = pk((oa.valid && r2a >= P.rmin2) ? ta : 0.f, (ob.valid && r2b >= P.rmin2) ? tb : 0.f);     // 0 for an empty slot
    unpk(mul2(fs, dx), oa.fx, ob.fx);
    unpk(mul2(fs, dy), oa.fy, ob.fy);
    unpk(mul2(fs, dz), oa.fz, ob.fz);
}
// Systolic schedule (topology.hpp): block b of the positions, one atom per lane for npos/2 rounds -- its position and its force
// sum stay in registers, the partners j = i + 1, i + 2, ... are read and updated in shared memory (consecutive lanes,
// consecutive positions: no bank conflicts), two rounds in flight.  gptr(off) = where the gradient words (+0, +32, +64) of the
// atom at block offset `off` live.  Returns the lane's energy sum.
template <bool GRAD, int NF, class GP>
__device__ __forceinline__ float pairs_systolic_block(const LigS& L, const ParDev& P, const float* blk, GP gptr, int b, int lane) {
    const int nblk = L.npos >> 5, K = L.npos >> 1;
    const int offi = b * 256 + lane;
    const float xi = blk[offi + kX], yi = blk[offi + kY], zi = blk[offi + kZ], qi = blk[offi + kQ];
    float fx = 0.f, fy = 0.f, fz = 0.f, ep = 0.f;
    const uint4* rec = L.pairs + b * 32 + lane;
    for (int k = 0; k < K; k += NF) {                    // K is a multiple of NF (npos = 128: 64)
        PairOut o[NF];
#pragma unroll
        for (int n = 0; n < NF; n += 2) pair_core2(P, rec[(k + n) * nblk * 32], rec[(k + n + 1) * nblk * 32], xi, yi, zi, qi, blk, o[n], o[n + 1]);
#pragma unroll
        for (int n = 0; n < NF; ++n) {
            if (GRAD) {                                  // an empty slot carries a zero force: no predicates on the updates
                float* g = gptr(o[n].oj);
                fx += o[n].fx; fy += o[n].fy; fz += o[n].fz; g[0] -= o[n].fx; g[32] -= o[n].fy; g[64] -= o[n].fz;
                __syncwarp();
            }
            ep += o[n].e;
        }
    }
    if (GRAD) {
        float* g = gptr(offi);
        g[0] += fx; g[32] += fy; g[64] += fz;
        __syncwarp();
    }
    return ep;
}
template <bool GRAD>
__device__ __forceinline__ float pair_apply(const WarpS& S, const PairOut& o) {
    if (GRAD) {
        float* pi = S.blk + o.oi, *pj = S.blk + o.oj;
        if (o.valid) { pi[kGX] += o.fx; pi[kGY] += o.fy; pi[kGZ] += o.fz; }
        __syncwarp();
        if (o.valid) { pj[kGX] -= o.fx; pj[kGY] -= o.fy; pj[kGZ] -= o.fz; }
        __syncwarp();
    }
    return o.e;
}
template <bool GRAD, bool MAYPAD>
__device__ __forceinline__ float pair_round(const LigS& L, const ParDev& P, const WarpS& S, int r, int lane) {
    return pair_apply<GRAD>(S, pair_compute<GRAD, MAYPAD>(L, P, S, r, lane));
}

// ---------------------------------------------------------------- full evaluation of one genotype by one warp
// Reads S.geno; writes S.grad (GRAD) and S.X; returns the total energy in every lane (NaN for |q|<1e-12).
template <bool GRAD>
__device__ __forceinline__ float eval_pose(const LigS& L, const GridDev& G, const ParDev& P, const WarpS& S, int lane,
                                           float& e_inter, float& e_intra) {
    const float tx = S.geno[0], ty = S.geno[1], tz = S.geno[2];
    float qw = S.geno[3], qx = S.geno[4], qy = S.geno[5], qz = S.geno[6];
    const float qn2 = qw * qw + qx * qx + qy * qy + qz * qz;
    if (!(qn2 >= 1e-24f)) {
        if (GRAD) for (int d = lane; d < 6 + L.R; d += 32) S.grad[d] = __int_as_float(0x7fc00000);
        e_inter = e_intra = __int_as_float(0x7fc00000);
        __syncwarp();
        return __int_as_float(0x7fc00000);
    }
    const float qi = 1.0f / sqrtf(qn2);
    qw *= qi; qx *= qi; qy *= qi; qz *= qi;
    const float r00 = 1.f - 2.f * (qy * qy + qz * qz), r01 = 2.f * (qx * qy - qw * qz), r02 = 2.f * (qx * qz + qw * qy);
    const float r10 = 2.f * (qx * qy + qw * qz), r11 = 1.f - 2.f * (qx * qx + qz * qz), r12 = 2.f * (qy * qz - qw * qx);
    const float r20 = 2.f * (qx * qz - qw * qy), r21 = 2.f * (qy * qz + qw * qx), r22 = 1.f - 2.f * (qx * qx + qy * qy);

    // (a1) sin/cos of every torsion, then per-fragment rigid transform T_f = T_root o Rot_k1 o ... o Rot_kd
    for (int f = lane; f < L.nfrag; f += 32) {
        float s = 0.f, c = 1.f;
        if (f > 0) sincosf(S.geno[7 + (L.fi[f].w >> 16)], &s, &c);
        S.sc[f] = make_float2(s, c);
    }
    __syncwarp();
    for (int f = lane; f < L.nfrag; f += 32) {
        float m00 = 1, m01 = 0, m02 = 0, m03 = 0, m10 = 0, m11 = 1, m12 = 0, m13 = 0, m20 = 0, m21 = 0, m22 = 1, m23 = 0;
        for (int cur = f; cur > 0; cur = L.fi[cur].x) {
            const float4 p0 = L.fg[2 * cur], u = L.fg[2 * cur + 1];
            const float2 sc = S.sc[cur];
            const float s = sc.x, c = sc.y, k = 1.f - c;
            const float a00 = fmaf(k * u.x, u.x, c), a01 = fmaf(k * u.x, u.y, -s * u.z), a02 = fmaf(k * u.x, u.z, s * u.y);
            const float a10 = fmaf(k * u.x, u.y, s * u.z), a11 = fmaf(k * u.y, u.y, c), a12 = fmaf(k * u.y, u.z, -s * u.x);
            const float a20 = fmaf(k * u.x, u.z, -s * u.y), a21 = fmaf(k * u.y, u.z, s * u.x), a22 = fmaf(k * u.z, u.z, c);
            // Rot(x) = A (x - p0) + p0 ; compose Rot o M
            float n00 = a00 * m00 + a01 * m10 + a02 * m20, n01 = a00 * m01 + a01 * m11 + a02 * m21,
                  n02 = a00 * m02 + a01 * m12 + a02 * m22;
            float n10 = a10 * m00 + a11 * m10 + a12 * m20, n11 = a10 * m01 + a11 * m11 + a12 * m21,
                  n12 = a10 * m02 + a11 * m12 + a12 * m22;
            float n20 = a20 * m00 + a21 * m10 + a22 * m20, n21 = a20 * m01 + a21 * m11 + a22 * m21,
                  n22 = a20 * m02 + a21 * m12 + a22 * m22;
            float dx = m03 - p0.x, dy = m13 - p0.y, dz = m23 - p0.z;
            float n03 = a00 * dx + a01 * dy + a02 * dz + p0.x, n13 = a10 * dx + a11 * dy + a12 * dz + p0.y,
                  n23 = a20 * dx + a21 * dy + a22 * dz + p0.z;
            m00 = n00; m01 = n01; m02 = n02; m03 = n03; m10 = n10; m11 = n11; m12 = n12; m13 = n13;
            m20 = n20; m21 = n21; m22 = n22; m23 = n23;
        }
        // T = Root o M, Root(y) = Rq y + t   (y already relative to the pivot)
        float t00 = r00 * m00 + r01 * m10 + r02 * m20, t01 = r00 * m01 + r01 * m11 + r02 * m21,
              t02 = r00 * m02 + r01 * m12 + r02 * m22, t03 = r00 * m03 + r01 * m13 + r02 * m23;
        float t10 = r10 * m00 + r11 * m10 + r12 * m20, t11 = r10 * m01 + r11 * m11 + r12 * m21,
              t12 = r10 * m02 + r11 * m12 + r12 * m22, t13 = r10 * m03 + r11 * m13 + r12 * m23;
        float t20 = r20 * m00 + r21 * m10 + r22 * m20, t21 = r20 * m01 + r21 * m11 + r22 * m21,
              t22 = r20 * m02 + r21 * m12 + r22 * m22, t23 = r20 * m03 + r21 * m13 + r22 * m23;
        S.fragT[3 * f] = make_float4(t00, t01, t02, t03 + tx);
        S.fragT[3 * f + 1] = make_float4(t10, t11, t12, t13 + ty);
        S.fragT[3 * f + 2] = make_float4(t20, t21, t22, t23 + tz);
        if (GRAD && f == 0) S.fragAx[1] = make_float4(0.f, 0.f, 0.f, 0.f);        // root pivot point = t
        if (GRAD && f > 0) {
            const float4 p0 = L.fg[2 * f], u = L.fg[2 * f + 1];
            S.fragAx[2 * f] = make_float4(t00 * u.x + t01 * u.y + t02 * u.z, t10 * u.x + t11 * u.y + t12 * u.z,
                                          t20 * u.x + t21 * u.y + t22 * u.z, 0.f);
            S.fragAx[2 * f + 1] = make_float4(t00 * p0.x + t01 * p0.y + t02 * p0.z + t03, t10 * p0.x + t11 * p0.y + t12 * p0.z + t13,
                                              t20 * p0.x + t21 * p0.y + t22 * p0.z + t23, 0.f);
        }
    }
    __syncwarp();

    // (a1,a2) atoms: pose, then trilinear lookup of the three maps
    // The rigid-body gradient (dE/dt, dE/domega) is summed from the GRID forces alone: intramolecular pair forces
    // cancel exactly in both (Newton's third law), so adding them would only put their rounding (r^-13 clash terms)
    // into two blocks they contribute nothing to.
    float eg = 0.f, rFx = 0.f, rFy = 0.f, rFz = 0.f, rTx = 0.f, rTy = 0.f, rTz = 0.f;
    for (int i = lane; i < L.npos; i += 32) {
        const uint32_t m = L.meta[i];
        if (m == 0xffffffffu) continue;                  // hole
        const float4 a = L.atoms[i];
        const int f = m >> 8;
        const float4 t0 = S.fragT[3 * f], t1 = S.fragT[3 * f + 1], t2 = S.fragT[3 * f + 2];
        const float x = fmaf(t0.x, a.x, fmaf(t0.y, a.y, fmaf(t0.z, a.z, t0.w)));
        const float y = fmaf(t1.x, a.x, fmaf(t1.y, a.y, fmaf(t1.z, a.z, t1.w)));
        const float z = fmaf(t2.x, a.x, fmaf(t2.y, a.y, fmaf(t2.z, a.z, t2.w)));
        float* b = S.blk + atom_slot_dev(i);
        b[kX] = x; b[kY] = y; b[kZ] = z; b[kQ] = a.w * P.elec_sqrt;
        float gx, gy, gz;
        eg += grid_atom<GRAD>(G, P, (int)(m & 0xff), a.w, x, y, z, gx, gy, gz);
        if (GRAD) {
            b[kGX] = gx; b[kGY] = gy; b[kGZ] = gz;
            const float rx = x - tx, ry = y - ty, rz = z - tz;
            rFx += gx; rFy += gy; rFz += gz;
            rTx += ry * gz - rz * gy; rTy += rz * gx - rx * gz; rTz += rx * gy - ry * gx;
        }
    }
    if (GRAD) {
        rFx = warp_sum(rFx); rFy = warp_sum(rFy); rFz = warp_sum(rFz);
        rTx = warp_sum(rTx); rTy = warp_sum(rTy); rTz = warp_sum(rTz);
    }
    __syncwarp();

    // (a3) intramolecular pairs: conflict-free warp rounds; the first nfull rounds have no padding slot
    float ep = 0.f;
    int r4 = 0;
    if (L.systolic) {                                   // one block of positions after the other, the lane's atom in registers
        for (int b = 0; b < (L.npos >> 5); ++b)
            ep += pairs_systolic_block<GRAD, 4>(L, P, S.blk, [&](int off) { return S.blk + off + kGX; }, b, lane);
        r4 = L.nrounds;
    }
    for (; r4 + 4 <= L.nfull; r4 += 4) {                // four rounds of arithmetic in flight, updates in round order
        const PairOut o0 = pair_compute<GRAD, false>(L, P, S, r4, lane), o1 = pair_compute<GRAD, false>(L, P, S, r4 + 1, lane),
                      o2 = pair_compute<GRAD, false>(L, P, S, r4 + 2, lane), o3 = pair_compute<GRAD, false>(L, P, S, r4 + 3, lane);
        ep += pair_apply<GRAD>(S, o0); ep += pair_apply<GRAD>(S, o1); ep += pair_apply<GRAD>(S, o2); ep += pair_apply<GRAD>(S, o3);
    }
    for (int r = r4; r < L.nfull; ++r) ep += pair_round<GRAD, false>(L, P, S, r, lane);
    for (int r = max(r4, L.nfull); r < L.nrounds; ++r) ep += pair_round<GRAD, true>(L, P, S, r, lane);
    e_inter = warp_sum(eg);
    e_intra = warp_sum(ep);

    // (a4) back-propagation: per-fragment force/torque, subtree sums, projection on the posed axes
    if (GRAD) {
        for (int f = lane; f < L.nfrag; f += 32) {
            const int4 ix = L.fi[f];
            const float4 pv = S.fragAx[2 * f + 1];               // this fragment's pivot point, relative to t
            const float px = tx + pv.x, py = ty + pv.y, pz = tz + pv.z;
            float Fx = 0, Fy = 0, Fz = 0, Tx = 0, Ty = 0, Tz = 0;
            for (int k = ix.y; k < ix.z; ++k) {
                const float* b = S.blk + atom_slot_dev(L.fragatoms[k]);
                const float gx = b[kGX], gy = b[kGY], gz = b[kGZ];
                const float rx = b[kX] - px, ry = b[kY] - py, rz = b[kZ] - pz;
                Fx += gx; Fy += gy; Fz += gz;
                Tx += ry * gz - rz * gy; Ty += rz * gx - rx * gz; Tz += rx * gy - ry * gx;
            }
            S.fragFT[2 * f] = make_float4(Fx, Fy, Fz, 0.f);
            S.fragFT[2 * f + 1] = make_float4(Tx, Ty, Tz, 0.f);
        }
        __syncwarp();
        for (int f = lane; f < L.nfrag; f += 32) {
            const int w = L.fi[f].w;
            const int sub_end = w & 0xffff;
            const float4 pf = S.fragAx[2 * f + 1];
            // force and torque ABOUT THIS fragment's pivot point of the whole subtree: each member's torque
            // (about its own pivot) is shifted by the short lever between the two pivots
            float Fx = 0, Fy = 0, Fz = 0, Tx = 0, Ty = 0, Tz = 0;
            for (int g = f; g < sub_end; ++g) {
                const float4 F = S.fragFT[2 * g], T = S.fragFT[2 * g + 1], pg = S.fragAx[2 * g + 1];
                const float lx = pg.x - pf.x, ly = pg.y - pf.y, lz = pg.z - pf.z;
                Fx += F.x; Fy += F.y; Fz += F.z;
                Tx += T.x + (ly * F.z - lz * F.y); Ty += T.y + (lz * F.x - lx * F.z); Tz += T.z + (lx * F.y - ly * F.x);
            }
            if (f == 0) {                               // rigid-body blocks: grid forces only (see the atom loop)
                S.grad[0] = rFx; S.grad[1] = rFy; S.grad[2] = rFz;
                S.grad[3] = rTx; S.grad[4] = rTy; S.grad[5] = rTz;
            } else {
                const float4 u = S.fragAx[2 * f];
                S.grad[6 + (w >> 16)] = u.x * Tx + u.y * Ty + u.z * Tz;
            }
        }
        __syncwarp();
    }
    return e_inter + e_intra;
}

// ---------------------------------------------------------------- Philox4x32-10 (R8)
__device__ __forceinline__ uint4 philox4x32_10(uint32_t k0, uint32_t k1, uint4 c) {
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c.x), l0 = 0xD2511F53u * c.x;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c.z), l1 = 0xCD9E8D57u * c.z;
        c = make_uint4(h1 ^ c.y ^ k0, l1, h0 ^ c.w ^ k1, l0);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}
enum : uint32_t { kInit = 0, kTournA = 1, kTournB = 2, kXover = 3, kMut = 4, kLsPick = 5, kSolisWets = 6 };
__device__ __forceinline__ uint4 draw4(unsigned long long seed, uint32_t draw, uint32_t purpose, uint32_t id, uint32_t gen) {
    return philox4x32_10((uint32_t)seed, (uint32_t)(seed >> 32), make_uint4(draw, purpose, id, gen));
}
__device__ __forceinline__ float u01(uint32_t x) { return (float)(x >> 8) * (1.0f / 16777216.0f); }
__device__ __forceinline__ int below(uint32_t x, int n) { return (int)(((unsigned long long)(x >> 8) * (unsigned)n) >> 24); }
__device__ __forceinline__ uint32_t pick_word(uint4 r, int w) { return w == 0 ? r.x : w == 1 ? r.y : w == 2 ? r.z : r.w; }

__device__ __forceinline__ float wrap_pi(float a) { return a - kTwoPi * floorf((a + kPi) * (1.0f / kTwoPi)); }

// q <- normalise((cos(th/2), sin(th/2) axis) (x) q) written to out[0..3]
__device__ __forceinline__ void rotate_quat(float cw, float ax, float ay, float az, const float* q, float* out) {
    const float n = 1.0f / sqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    const float w = q[0] * n, x = q[1] * n, y = q[2] * n, z = q[3] * n;
    float ow = cw * w - ax * x - ay * y - az * z;
    float oxx = cw * x + ax * w + ay * z - az * y;
    float oy = cw * y - ax * z + ay * w + az * x;
    float oz = cw * z + ax * y - ay * x + az * w;
    const float m = 1.0f / sqrtf(ow * ow + oxx * oxx + oy * oy + oz * oz);
    out[0] = ow * m; out[1] = oxx * m; out[2] = oy * m; out[3] = oz * m;
}

// ---------------------------------------------------------------- GA operators (R9), one warp per individual
__device__ inline void ga_init_individual(const GridDev& G, int R, unsigned long long seed, uint32_t id, float* geno, int lane) {
    if (lane < 3) {
        const uint4 r = draw4(seed, 0, kInit, id, 0);
        const float u = u01(pick_word(r, lane));
        geno[lane] = lane == 0 ? fmaf(u, G.bx, G.ox) : lane == 1 ? fmaf(u, G.by, G.oy) : fmaf(u, G.bz, G.oz);
    } else if (lane == 3) {
        const uint4 r = draw4(seed, 1, kInit, id, 0);
        const float u1 = u01(r.x), u2 = u01(r.y), u3 = u01(r.z);
        const float s1 = sqrtf(1.f - u1), s2 = sqrtf(u1);
        float sa, ca, sb, cb;
        sincospif(2.f * u2, &sa, &ca);
        sincospif(2.f * u3, &sb, &cb);
        geno[3] = s2 * cb; geno[4] = s1 * sa; geno[5] = s1 * ca; geno[6] = s2 * sb;
    }
    for (int k = lane; k < R; k += 32) {
        const uint4 r = draw4(seed, 2 + k / 4, kInit, id, 0);
        geno[7 + k] = fmaf(u01(pick_word(r, k & 3)), kTwoPi, -kPi);
    }
}

__device__ __forceinline__ int tournament(const ParDev& P, int Pn, const float* E, unsigned long long seed, uint32_t purpose,
                                          uint32_t id, uint32_t gen, int* dec) {
    const uint4 r = draw4(seed, 0, purpose, id, gen);
    const int s1 = below(r.x, Pn), s2 = below(r.y, Pn);
    const bool first = E[s1] <= E[s2];
    const int lo = first ? s1 : s2, hi = first ? s2 : s1;
    const int pick = (u01(r.z) < P.tourn_prob) ? lo : hi;
    if (dec) { dec[0] = s1; dec[1] = s2; dec[2] = pick; }
    return pick;
}

// child of slot s>=1 written to geno (shared, [7+R]); all lanes call; dec (global, 10 ints) optional
__device__ inline void ga_make_child(const ParDev& P, int Pn, int R, unsigned long long seed, uint32_t id, uint32_t gen,
                                     const float* pop, const float* E, float* geno, int* dec, int lane) {
    const int Gn = 7 + R, NB = 4 + R;
    int* d0 = (dec && lane == 0) ? dec : nullptr;
    const int A = tournament(P, Pn, E, seed, kTournA, id, gen, d0);
    const int B = tournament(P, Pn, E, seed, kTournB, id, gen, d0 ? d0 + 3 : nullptr);
    const uint4 rx = draw4(seed, 0, kXover, id, gen);
    const int c1 = below(rx.y, NB + 1), c2 = below(rx.z, NB + 1);
    const int p1 = min(c1, c2), p2 = max(c1, c2);
    const bool xo = u01(rx.x) < P.xover_rate;
    if (d0) { d0[6] = xo; d0[7] = p1; d0[8] = p2; }
    const float* gA = pop + (size_t)A * Gn;
    const float* gB = pop + (size_t)B * Gn;
    unsigned mutmask = 0;
    for (int b0 = 0; b0 < NB; b0 += 32) {
        const int b = b0 + lane;
        bool mut = false;
        if (b < NB) {
            const float* src = (xo && b >= p1 && b < p2) ? gB : gA;
            const uint4 rm = draw4(seed, (uint32_t)b, kMut, id, gen);
            mut = u01(rm.x) < P.mut_rate;
            const float amt = 2.f * u01(rm.y) - 1.f;
            if (b < 3) {
                geno[b] = mut ? src[b] + amt * P.dmov : src[b];
            } else if (b == 3) {
                if (mut) {
                    const float ang = amt * P.dang, z = 2.f * u01(rm.z) - 1.f;
                    const float sxy = sqrtf(fmaxf(0.f, 1.f - z * z));
                    float sp, cp, sh, ch;
                    sincospif(2.f * u01(rm.w), &sp, &cp);
                    sincosf(0.5f * ang, &sh, &ch);
                    const float q[4] = {src[3], src[4], src[5], src[6]};
                    float o[4];
                    rotate_quat(ch, sh * sxy * cp, sh * sxy * sp, sh * z, q, o);
                    geno[3] = o[0]; geno[4] = o[1]; geno[5] = o[2]; geno[6] = o[3];
                } else {
                    geno[3] = src[3]; geno[4] = src[4]; geno[5] = src[5]; geno[6] = src[6];
                }
            } else {
                const int gi = 4 + b - 1;
                geno[gi] = mut ? wrap_pi(src[gi] + amt * P.dang) : src[gi];
            }
        }
        const unsigned bal = __ballot_sync(kFull, mut);
        if (b0 == 0) mutmask = bal & 0x7fffffffu;
    }
    if (d0) d0[9] = (int)mutmask;
    __syncwarp();
}

// The same child, made by ONE thread straight into global memory (dock_ga_lane_kernel: a thread per individual of the
// new population).  Same draws (counter = gene block, purpose, individual, generation) and the same expressions per
// gene block as ga_make_child, so the integer decisions and the genotypes are identical bit for bit.
__device__ inline void ga_make_child_thread(const ParDev& P, int Pn, int R, unsigned long long seed, uint32_t id, uint32_t gen,
                                            const float* pop, const float* E, float* geno, int* dec) {
    const int Gn = 7 + R, NB = 4 + R;
    const int A = tournament(P, Pn, E, seed, kTournA, id, gen, dec);
    const int B = tournament(P, Pn, E, seed, kTournB, id, gen, dec ? dec + 3 : nullptr);
    const uint4 rx = draw4(seed, 0, kXover, id, gen);
    const int c1 = below(rx.y, NB + 1), c2 = below(rx.z, NB + 1);
    const int p1 = min(c1, c2), p2 = max(c1, c2);
    const bool xo = u01(rx.x) < P.xover_rate;
    if (dec) { dec[6] = xo; dec[7] = p1; dec[8] = p2; }
    const float* gA = pop + (size_t)A * Gn;
    const float* gB = pop + (size_t)B * Gn;
    unsigned mutmask = 0;
    for (int b = 0; b < NB; ++b) {
        const float* src = (xo && b >= p1 && b < p2) ? gB : gA;
        const uint4 rm = draw4(seed, (uint32_t)b, kMut, id, gen);
        const bool mut = u01(rm.x) < P.mut_rate;
        const float amt = 2.f * u01(rm.y) - 1.f;
        if (b < 3) {
            geno[b] = mut ? src[b] + amt * P.dmov : src[b];
        } else if (b == 3) {
            if (mut) {
                const float ang = amt * P.dang, z = 2.f * u01(rm.z) - 1.f;
                const float sxy = sqrtf(fmaxf(0.f, 1.f - z * z));
                float sp, cp, sh, ch;
                sincospif(2.f * u01(rm.w), &sp, &cp);
                sincosf(0.5f * ang, &sh, &ch);
                const float q[4] = {src[3], src[4], src[5], src[6]};
                float o[4];
                rotate_quat(ch, sh * sxy * cp, sh * sxy * sp, sh * z, q, o);
                geno[3] = o[0]; geno[4] = o[1]; geno[5] = o[2]; geno[6] = o[3];
            } else {
                geno[3] = src[3]; geno[4] = src[4]; geno[5] = src[5]; geno[6] = src[6];
            }
        } else {
            const int gi = 4 + b - 1;
            geno[gi] = mut ? wrap_pi(src[gi] + amt * P.dang) : src[gi];
        }
        if (mut && b < 31) mutmask |= 1u << b;
    }
    if (dec) dec[9] = (int)mutmask;
}

// ---------------------------------------------------------------- full evaluation of one genotype by a TEAM of W warps
// One team of kTeamW warps per individual (one or four teams per CTA, sharing the ligand image), threads over atoms and pairs: for launches with so few chains that one warp per
// chain leaves most schedulers idle (a single ligand: 180 chains on 592 schedulers), the evaluation itself is split.
// The 32 W threads take one atom each (pose, grid lookup); warp w takes the pair rounds r = w (mod W), several rounds in flight, and adds their forces into its own gradient plane (W planes of gx|gy|gz, 96
// floats per 32 atoms, in T.gpl), so no two warps ever update the same word; the atom's thread sums the planes in a fixed
// order.  Same arithmetic as eval_pose; the summation order differs (fixed, so results are reproducible).
constexpr int kTeamW = 4;
__host__ __device__ inline int team_scratch_floats(int N, int nfrag, int R) {
    return warp_scratch_floats(N, nfrag, R) + kTeamW * ((N + 31) / 32) * 96 + 8 * kTeamW + 8 + 24 * nfrag + pad4(7 + R) + 4 * pad4(6 + R);
}
// red: per warp w [8w .. 8w+8) = partial (e_grid, e_pairs, grid force F(3), grid torque about t T(3)); [8 kTeamW] = the
// "every gradient component was finite" flag.
// The ADADELTA chain keeps TWO copies of what a step changes, used alternately: the genotype (S.geno | geno1), the optimiser
// state ad[b] = E[g^2](Dpad) | E[dx^2](Dpad), and the local transforms lt[b]: fragment f > 0 (rotation A by its torsion angle
// about its axis through p0: x -> A (x - p0) + p0) as three rows (A_r, p0_r) at lt[b][3f + r]; slot 0 holds the rows of the
// rigid-body rotation (w = 0).  While copy b is being evaluated the step to the next point is written into copy b ^ 1.
struct TeamS {
    WarpS S;
    float* gpl; float* red; float* geno1; float* ad0; float4* lt0;     // copy b of the state at ad0 + b * 2 Dpad, of the transforms at lt0 + b * 3 nfrag
    int wi, gplane, bar;                                // gplane = floats per plane; bar = the team's named barrier
};
__device__ inline TeamS team_view(float* base, const LigS& L, int wi) {
    TeamS T;
    T.S = warp_view(base, L);
    T.gpl = T.S.blk + (L.npos / 32) * 256;
    T.red = T.gpl + kTeamW * (L.npos / 32) * 96;
    T.lt0 = reinterpret_cast<float4*>(T.red + 8 * kTeamW + 8);
    T.geno1 = reinterpret_cast<float*>(T.lt0 + 6 * L.nfrag);
    T.ad0 = T.geno1 + pad4(7 + L.R);
    T.wi = wi; T.gplane = (L.npos / 32) * 96; T.bar = 1;
    return T;
}
// eval_pose's rotation about the torsion axis, for (sin, cos) of the angle
__device__ __forceinline__ void team_local_transform(const LigS& L, float4* lt, int f, float s, float c) {
    const float4 p0 = L.fg[2 * f], u = L.fg[2 * f + 1];
    const float k = 1.f - c;
    const float a00 = fmaf(k * u.x, u.x, c), a01 = fmaf(k * u.x, u.y, -s * u.z), a02 = fmaf(k * u.x, u.z, s * u.y);
    const float a10 = fmaf(k * u.x, u.y, s * u.z), a11 = fmaf(k * u.y, u.y, c), a12 = fmaf(k * u.y, u.z, -s * u.x);
    const float a20 = fmaf(k * u.x, u.z, -s * u.y), a21 = fmaf(k * u.y, u.z, s * u.x), a22 = fmaf(k * u.z, u.z, c);
    lt[3 * f] = make_float4(a00, a01, a02, p0.x);
    lt[3 * f + 1] = make_float4(a10, a11, a12, p0.y);
    lt[3 * f + 2] = make_float4(a20, a21, a22, p0.z);
}
// eval_pose's rotation matrix of the (re-normalised) quaternion q[4]
__device__ __forceinline__ void team_rotation(float4* lt, const float* q) {
    float qw = q[0], qx = q[1], qy = q[2], qz = q[3];
    const float qi = 1.0f / sqrtf(qw * qw + qx * qx + qy * qy + qz * qz);
    qw *= qi; qx *= qi; qy *= qi; qz *= qi;
    lt[0] = make_float4(1.f - 2.f * (qy * qy + qz * qz), 2.f * (qx * qy - qw * qz), 2.f * (qx * qz + qw * qy), 0.f);
    lt[1] = make_float4(2.f * (qx * qy + qw * qz), 1.f - 2.f * (qx * qx + qz * qz), 2.f * (qy * qz - qw * qx), 0.f);
    lt[2] = make_float4(2.f * (qx * qz - qw * qy), 2.f * (qy * qz + qw * qx), 1.f - 2.f * (qx * qx + qy * qy), 0.f);
}
__device__ __forceinline__ void team_sync(const TeamS& T) { asm volatile("bar.sync %0, %1;" ::"r"(T.bar), "n"(kTeamW * 32) : "memory"); }
// index in a plane of the atom at blk offset `off` (256 floats per 32 atoms -> 96): words +0, +32, +64
__device__ __forceinline__ int plane_index(int off) { return off - (off >> 8) * 160; }
template <bool MAYPAD>
__device__ __forceinline__ void team_pair_apply(float* plane, const PairOut& o) {
    float* gi = plane + plane_index(o.oi), *gj = plane + plane_index(o.oj);
    if (!MAYPAD || o.valid) { gi[0] += o.fx; gi[32] += o.fy; gi[64] += o.fz; }
    __syncwarp();
    if (!MAYPAD || o.valid) { gj[0] -= o.fx; gj[32] -= o.fy; gj[64] -= o.fz; }
    __syncwarp();
}

// Evaluation of copy b of the chain's point up to the per-atom gradients: pose, pairs, lookups (a1-a3 and the grid part of
// a4).  On return (after a team barrier) S.blk holds positions and summed per-atom gradients, T.red the warps' partial
// energies and rigid-body sums.  Returns the energy in every thread; NaN, before any barrier, for |q| < 1e-12.
// NF: full pair rounds in flight per warp (registers); SYS: knows the systolic pair schedule
template <int NF, bool SYS>
__device__ __forceinline__ float team_front(const LigS& L, const GridDev& G, const ParDev& P, const TeamS& T, int lane, int b,
                                            float& e_inter, float& e_intra) {
    constexpr bool GRAD = true;
    const WarpS& S = T.S;
    const int wi = T.wi;
    const float* geno = b ? T.geno1 : S.geno;
    const float4* lt = T.lt0 + b * 3 * L.nfrag;
    const float tx = geno[0], ty = geno[1], tz = geno[2];
    {
        const float qw = geno[3], qx = geno[4], qy = geno[5], qz = geno[6];
        const float qn2 = qw * qw + qx * qx + qy * qy + qz * qz;
        if (!(qn2 >= 1e-24f)) {                         // the same in every thread of the team
            e_inter = e_intra = __int_as_float(0x7fc00000);
            return __int_as_float(0x7fc00000);
        }
    }
    // (a1) pose: a thread per atom carries the atom's reference position through the local transforms of its fragment and of
    // the fragment's ancestors (left in shared memory by the step that led here: team_local_transform), then through the
    // rigid-body rotation (team_rotation) and the translation; it asks for the atom's two map sectors and clears the atom's
    // gradient planes.  Two more threads per fragment f > 0 carry its axis (a direction) and its pivot (a point, kept
    // relative to t) the same way, for the torsion gradients.  eval_pose's transforms applied one after the other instead of
    // composed first.
    {
        const float4 R0 = lt[0], R1 = lt[1], R2 = lt[2];
        const int nitem = L.npos + 2 * L.nfrag;
        for (int it = wi * 32 + lane; it < nitem; it += 32 * kTeamW) {
            const bool atom = it < L.npos;
            uint32_t m = 0;
            float4 v;
            int f;
            bool pt = true;
            if (atom) {
                m = L.meta[it];
                if (m == 0xffffffffu) continue;          // hole
                v = L.atoms[it];
                f = m >> 8;
            } else {
                f = (it - L.npos) >> 1;
                if (f == 0) continue;
                pt = (it - L.npos) & 1;
                v = L.fg[2 * f + (pt ? 0 : 1)];
            }
            float vx = v.x, vy = v.y, vz = v.z;
            for (int cur = f; cur > 0;) {
                const float4 a0 = lt[3 * cur], a1 = lt[3 * cur + 1], a2 = lt[3 * cur + 2];
                cur = L.fi[cur].x;
                const float dx = pt ? vx - a0.w : vx, dy = pt ? vy - a1.w : vy, dz = pt ? vz - a2.w : vz;
                vx = a0.x * dx + a0.y * dy + a0.z * dz + (pt ? a0.w : 0.f);
                vy = a1.x * dx + a1.y * dy + a1.z * dz + (pt ? a1.w : 0.f);
                vz = a2.x * dx + a2.y * dy + a2.z * dz + (pt ? a2.w : 0.f);
            }
            const float wx = R0.x * vx + R0.y * vy + R0.z * vz, wy = R1.x * vx + R1.y * vy + R1.z * vz,
                        wz = R2.x * vx + R2.y * vy + R2.z * vz;
            if (atom) {
                const float x = wx + tx, y = wy + ty, z = wz + tz;
                const int off = atom_slot_dev(it);
                float* b = S.blk + off;
                b[kX] = x; b[kY] = y; b[kZ] = z; b[kQ] = v.w * P.elec_sqrt;
                grid_prefetch(G, grid_cell(G, (int)(m & 0xff), x, y, z));
                float* g = T.gpl + plane_index(off);
#pragma unroll
                for (int w = 0; w < kTeamW; ++w) { g[w * T.gplane] = 0.f; g[w * T.gplane + 32] = 0.f; g[w * T.gplane + 64] = 0.f; }
            } else {
                S.fragAx[2 * f + (pt ? 1 : 0)] = make_float4(wx, wy, wz, 0.f);
            }
        }
    }
    team_sync(T);

    // (a3) intramolecular pairs: warp wi takes rounds wi, wi + W, ...; forces go to plane wi.  NF full rounds at a time:
    // their arithmetic is independent of the force updates, which follow in round order.
    float ep = 0.f;
    float* plane = T.gpl + wi * T.gplane;
    int r = wi;
    if (SYS && L.systolic) {                            // block wi of the positions (npos / 32 = kTeamW), the thread's atom in registers
        ep = pairs_systolic_block<GRAD, NF>(L, P, S.blk, [&](int off) { return plane + plane_index(off); }, wi, lane);
        r = L.nrounds;
    }
    for (; r + (NF - 1) * kTeamW < L.nfull; r += NF * kTeamW) {
        PairOut o[NF];
#pragma unroll
        for (int k = 0; k < NF; ++k) o[k] = pair_compute<GRAD, false>(L, P, S, r + k * kTeamW, lane);
#pragma unroll
        for (int k = 0; k < NF; ++k) {
            if (GRAD) team_pair_apply<false>(plane, o[k]);
            ep += o[k].e;
        }
    }
    if (NF > 2)
        for (; r + kTeamW < L.nfull; r += 2 * kTeamW) {
            const PairOut o0 = pair_compute<GRAD, false>(L, P, S, r, lane), o1 = pair_compute<GRAD, false>(L, P, S, r + kTeamW, lane);
            if (GRAD) { team_pair_apply<false>(plane, o0); team_pair_apply<false>(plane, o1); }
            ep += o0.e; ep += o1.e;
        }
    for (; r < L.nrounds; r += kTeamW) {
        const PairOut o = pair_compute<GRAD, true>(L, P, S, r, lane);
        if (GRAD) team_pair_apply<true>(plane, o);
        ep += o.e;
    }
    team_sync(T);

    // (a2) trilinear lookups, after the pairs so that the sectors asked for in (a1) have arrived: a thread per atom looks the
    // atom up and adds the planes to the grid gradient (fixed order grid+0+1+2+3).
    float red[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};      // e_grid, e_pairs, rigid-body sums F(3), T(3): grid forces only (eval_pose)
    for (int i = wi * 32 + lane; i < L.npos; i += 32 * kTeamW) {
        const uint32_t m = L.meta[i];
        if (m == 0xffffffffu) continue;
        const int off = atom_slot_dev(i);
        float* b = S.blk + off;
        const float x = b[kX], y = b[kY], z = b[kZ];
        float gx, gy, gz;
        red[0] += grid_atom_l1<GRAD>(G, P, (int)(m & 0xff), L.atoms[i].w, x, y, z, gx, gy, gz);
        if (GRAD) {
            const float rx = x - tx, ry = y - ty, rz = z - tz;
            red[2] += gx; red[3] += gy; red[4] += gz;
            red[5] += ry * gz - rz * gy; red[6] += rz * gx - rx * gz; red[7] += rx * gy - ry * gx;
            const float* g = T.gpl + plane_index(off);
#pragma unroll
            for (int w = 0; w < kTeamW; ++w) { gx += g[w * T.gplane]; gy += g[w * T.gplane + 32]; gz += g[w * T.gplane + 64]; }
            b[kGX] = gx; b[kGY] = gy; b[kGZ] = gz;
        }
    }
    red[1] = ep;
    const float part = warp_sum8(red, lane);
    if ((lane & 3) == 0) T.red[8 * wi + (lane >> 2)] = part;
    team_sync(T);
    e_inter = 0.f; e_intra = 0.f;
#pragma unroll
    for (int w = 0; w < kTeamW; ++w) { e_inter += T.red[8 * w]; e_intra += T.red[8 * w + 1]; }

    return e_inter + e_intra;
}

// ---------------------------------------------------------------- ADADELTA local search (R7), one warp
// Start genotype in S.geno; on return S.best holds the best genotype seen and the function returns its
// energy (the carried energy e_start if no finite evaluation happened).  iters = evaluations performed.
__device__ inline float adadelta_search(const LigS& L, const GridDev& G, const ParDev& P, const WarpS& S, int lane,
                                        float e_start, int& iters, float* trace = nullptr) {
    const int R = L.R, D = 6 + R, Gn = 7 + R;
    float Eg2[3] = {0.f, 0.f, 0.f}, Ed2[3] = {0.f, 0.f, 0.f};         // component d = lane + 32*c  (D <= 70)
    float bestE = __int_as_float(0x7f800000);
    for (int d = lane; d < Gn; d += 32) S.best[d] = S.geno[d];
    __syncwarp();
    int it = 0;
    while (it < P.lsit) {
        float ei, ea;
        const float e = eval_pose<true>(L, G, P, S, lane, ei, ea);
        if (trace && lane == 0) trace[it] = e;
        ++it;
        bool ok = isfinite(e);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int d = lane + 32 * c;
            if (d < D) ok = ok && isfinite(S.grad[d]);
        }
        if (!__all_sync(kFull, ok)) break;
        if (e < bestE) {
            bestE = e;
            for (int d = lane; d < Gn; d += 32) S.best[d] = S.geno[d];
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int d = lane + 32 * c;
            if (d < D) {
                const float g = S.grad[d];
                Eg2[c] = P.ad_rho * Eg2[c] + (1.f - P.ad_rho) * g * g;
                const float dl = -(sqrtf(Ed2[c] + P.ad_eps) / sqrtf(Eg2[c] + P.ad_eps)) * g;
                Ed2[c] = P.ad_rho * Ed2[c] + (1.f - P.ad_rho) * dl * dl;
                S.grad[d] = dl;
            }
        }
        __syncwarp();
        // apply the step: t += dt ; q <- normalise(exp(dw/2) (x) q) ; tau <- wrap(tau + dtau)
        float newv[3];
        float newq[4];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int gI = lane + 32 * c;
            if (gI < 3) newv[c] = S.geno[gI] + S.grad[gI];
            else if (gI >= 7 && gI < Gn) newv[c] = wrap_pi(S.geno[gI] + S.grad[gI - 1]);
        }
        if (lane == 3) {
            const float wx = S.grad[3], wy = S.grad[4], wz = S.grad[5];
            const float th = sqrtf(wx * wx + wy * wy + wz * wz);
            float sh, ch;
            sincosf(0.5f * th, &sh, &ch);
            const float k = th > 1e-12f ? sh / th : 0.5f;
            rotate_quat(ch, k * wx, k * wy, k * wz, S.geno + 3, newq);
        }
        __syncwarp();
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int gI = lane + 32 * c;
            if (gI < 3 || (gI >= 7 && gI < Gn)) S.geno[gI] = newv[c];
        }
        if (lane == 3) { S.geno[3] = newq[0]; S.geno[4] = newq[1]; S.geno[5] = newq[2]; S.geno[6] = newq[3]; }
        __syncwarp();
    }
    iters = it;
    return isfinite(bestE) ? bestE : e_start;
}

// ---------------------------------------------------------------- ADADELTA local search (R7), one team
// adadelta_search with the evaluation spread over the team and the step computed where its gradient component appears,
// before anyone knows whether the iteration counts: while copy b of (genotype, optimiser state, local transforms) is being
// evaluated, the step to the next point goes into copy b ^ 1 -- the translation and rotation components (lanes 0..5 of the
// last warp: gradient = the warps' grid-force sums, known after the lookups; lane 3 builds the quaternion and its rotation
// matrix) alongside the torsion gradients (eight lanes per torsion over the atoms of its subtree: u . ((r - pivot) x g), eval_pose's
// terms in another, fixed order; the lane that holds the sum steps the angle and leaves the fragment's local transform).  One
// barrier later every thread sees the energy and the "all finite" flag and takes the same decision: stop, or note the
// evaluated point as the best so far and move on to copy b ^ 1.  Five team barriers per iteration.
// Called by all kTeamW warps with S.geno ready and visible; S.best holds the result.
__device__ __forceinline__ float adadelta_step(const ParDev& P, float g, const float* st, float* st_next, int d, int Dp) {
    const float Eg2 = P.ad_rho * st[d] + (1.f - P.ad_rho) * g * g;
    const float dl = -(sqrtf(st[Dp + d] + P.ad_eps) / sqrtf(Eg2 + P.ad_eps)) * g;
    st_next[d] = Eg2;
    st_next[Dp + d] = P.ad_rho * st[Dp + d] + (1.f - P.ad_rho) * dl * dl;
    return dl;
}
template <int NF, bool SYS = false>
__device__ inline float adadelta_search_team(const LigS& L, const GridDev& G, const ParDev& P, const TeamS& T, int lane, float e_start,
                                             int& iters, float* trace = nullptr) {
    const WarpS& S = T.S;
    const int R = L.R, Gn = 7 + R, Dp = pad4(6 + R), wi = T.wi, tid = wi * 32 + lane;
    float bestE = __int_as_float(0x7f800000);
    for (int d = tid; d < Gn; d += 32 * kTeamW) S.best[d] = S.geno[d];
    for (int d = tid; d < 2 * Dp; d += 32 * kTeamW) T.ad0[d] = 0.f;
    for (int f = 1 + tid; f < L.nfrag; f += 32 * kTeamW) {
        float s, c;
        sincosf(S.geno[7 + (L.fi[f].w >> 16)], &s, &c);
        team_local_transform(L, T.lt0, f, s, c);
    }
    if (tid == 32 * (kTeamW - 1)) team_rotation(T.lt0, S.geno + 3);
    float* flag = T.red + 8 * kTeamW;                   // "every gradient component so far was finite": cleared by the thread that sees otherwise
    if (tid == 31) *flag = 1.f;
    team_sync(T);
    int it = 0, b = 0;
    while (it < P.lsit) {
        float ei, ea;
        const float e = team_front<NF, SYS>(L, G, P, T, lane, b, ei, ea);         // ends with a team barrier (unless NaN: |q| ~ 0)
        if (trace && tid == 0) trace[it] = e;
        ++it;
        if (!isfinite(e)) break;                         // the same in every thread
        const float* geno = b ? T.geno1 : S.geno;
        float* gnext = b ? S.geno : T.geno1;
        const float* st = T.ad0 + b * 2 * Dp;
        float* st_next = T.ad0 + (b ^ 1) * 2 * Dp;
        float4* lt_next = T.lt0 + (b ^ 1) * 3 * L.nfrag;
        if (wi == kTeamW - 1) {                         // rigid-body blocks: the warps' grid-force sums, fixed order
            float dl = 0.f;
            if (lane < 6) {
                float v = T.red[2 + lane];
#pragma unroll
                for (int w = 1; w < kTeamW; ++w) v += T.red[8 * w + 2 + lane];
                if (!isfinite(v)) *flag = 0.f;
                dl = adadelta_step(P, v, st, st_next, lane, Dp);
                if (lane < 3) gnext[lane] = geno[lane] + dl;
            }
            const float wx = __shfl_sync(kFull, dl, 3), wy = __shfl_sync(kFull, dl, 4), wz = __shfl_sync(kFull, dl, 5);
            if (lane == 3) {                            // q <- normalise(exp(dw/2) (x) q)
                float newq[4];
                const float th = sqrtf(wx * wx + wy * wy + wz * wz);
                float sh, ch;
                sincosf(0.5f * th, &sh, &ch);
                const float k = th > 1e-12f ? sh / th : 0.5f;
                rotate_quat(ch, k * wx, k * wy, k * wz, geno + 3, newq);
                gnext[3] = newq[0]; gnext[4] = newq[1]; gnext[5] = newq[2]; gnext[6] = newq[3];
                team_rotation(lt_next, newq);
            }
        }
        {
            const float tx = geno[0], ty = geno[1], tz = geno[2];
            const int nitem = 8 * (L.nfrag - 1);
            for (int base = wi * 32; base < nitem; base += 32 * kTeamW) {
                const int item = base + lane, f = 1 + (item >> 3);
                float v0 = 0.f, v1 = 0.f;
                int w = 0;
                if (item < nitem) {
                    const int4 ix = L.fi[f];
                    w = ix.w;
                    const int kend = L.fi[(w & 0xffff) - 1].z;
                    const float4 u = S.fragAx[2 * f], pv = S.fragAx[2 * f + 1];
                    const float px = tx + pv.x, py = ty + pv.y, pz = tz + pv.z;
                    int k = ix.y + (item & 7);
                    for (; k + 8 < kend; k += 16) {
                        const float* b0 = S.blk + atom_slot_dev(L.fragatoms[k]), *b1 = S.blk + atom_slot_dev(L.fragatoms[k + 8]);
                        const float gx0 = b0[kGX], gy0 = b0[kGY], gz0 = b0[kGZ], rx0 = b0[kX] - px, ry0 = b0[kY] - py, rz0 = b0[kZ] - pz;
                        const float gx1 = b1[kGX], gy1 = b1[kGY], gz1 = b1[kGZ], rx1 = b1[kX] - px, ry1 = b1[kY] - py, rz1 = b1[kZ] - pz;
                        v0 += u.x * (ry0 * gz0 - rz0 * gy0) + u.y * (rz0 * gx0 - rx0 * gz0) + u.z * (rx0 * gy0 - ry0 * gx0);
                        v1 += u.x * (ry1 * gz1 - rz1 * gy1) + u.y * (rz1 * gx1 - rx1 * gz1) + u.z * (rx1 * gy1 - ry1 * gx1);
                    }
                    if (k < kend) {
                        const float* b0 = S.blk + atom_slot_dev(L.fragatoms[k]);
                        const float gx0 = b0[kGX], gy0 = b0[kGY], gz0 = b0[kGZ], rx0 = b0[kX] - px, ry0 = b0[kY] - py, rz0 = b0[kZ] - pz;
                        v0 += u.x * (ry0 * gz0 - rz0 * gy0) + u.y * (rz0 * gx0 - rx0 * gz0) + u.z * (rx0 * gy0 - ry0 * gx0);
                    }
                }
                float v = v0 + v1;
                v += __shfl_xor_sync(kFull, v, 4); v += __shfl_xor_sync(kFull, v, 2); v += __shfl_xor_sync(kFull, v, 1);
                if (item < nitem && (item & 7) == 0) {  // the torsion's gradient: step the angle, leave the local transform
                    const int ti = w >> 16;
                    if (!isfinite(v)) *flag = 0.f;
                    const float dl = adadelta_step(P, v, st, st_next, 6 + ti, Dp);
                    const float nv = wrap_pi(geno[7 + ti] + dl);
                    gnext[7 + ti] = nv;
                    float sn, cs;
                    sincosf(nv, &sn, &cs);
                    team_local_transform(L, lt_next, f, sn, cs);
                }
            }
        }
        team_sync(T);                                    // the step, the flag
        if (*flag == 0.f) break;                         // the same in every thread
        if (e < bestE) {
            bestE = e;
            for (int d = tid; d < Gn; d += 32 * kTeamW) S.best[d] = geno[d];     // copy b is not written again before four more barriers
        }
        b ^= 1;
    }
    iters = it;
    return isfinite(bestE) ? bestE : e_start;
}

// ---------------------------------------------------------------- Solis-Wets local search (R11), one warp
// Start genotype in S.geno with carried energy e_start (not re-evaluated).  Per iteration: delta = rho*amp*(2u-1) + bias
// (u: Philox word d&3 of draw (it*ceil(D/4) + d/4, kSolisWets, id, gen)); x (+) delta is tried, then x (-) delta; a
// strictly better trial is accepted and pulls the bias its way, a double failure halves the bias; sw_max_succ
// successes in a row expand rho, sw_max_fail failures contract it; ends at lsit iterations or rho < sw_rho_lb.
// On return S.best holds the accepted genotype; returns its energy; evals = evaluations performed.
__device__ inline float solis_wets_search(const LigS& L, const GridDev& G, const ParDev& P, const WarpS& S, int lane, float e_start,
                                          unsigned long long seed, uint32_t id, uint32_t gen, int& evals, float* trace = nullptr) {
    const int R = L.R, D = 6 + R, Gn = 7 + R, nq = (D + 3) / 4;
    float bias[3] = {0.f, 0.f, 0.f}, delta[3] = {0.f, 0.f, 0.f};      // component d = lane + 32*c  (D <= 70)
    for (int d = lane; d < Gn; d += 32) S.best[d] = S.geno[d];
    __syncwarp();
    float E = e_start, rho = P.sw_rho0;
    int ns = 0, nf = 0, it = 0;
    evals = 0;
    while (it < P.lsit && !(rho < P.sw_rho_lb)) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int d = lane + 32 * c;
            if (d < D) {
                const uint4 r = draw4(seed, (uint32_t)(it * nq + (d >> 2)), kSolisWets, id, gen);
                const float xi = 2.f * u01(pick_word(r, d & 3)) - 1.f;
                delta[c] = rho * (d < 3 ? P.dmov : P.dang) * xi + bias[c];
            }
        }
        bool ok = false;
        float e = E;
        for (int trial = 0; trial < 2 && !ok; ++trial) {
            const float sg = trial ? -1.f : 1.f;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const int d = lane + 32 * c;
                if (d < D) S.grad[d] = sg * delta[c];
            }
            __syncwarp();
            for (int gI = lane; gI < Gn; gI += 32) {
                if (gI < 3) S.geno[gI] = S.best[gI] + S.grad[gI];
                else if (gI >= 7) S.geno[gI] = wrap_pi(S.best[gI] + S.grad[gI - 1]);
            }
            if (lane == 3) {
                const float wx = S.grad[3], wy = S.grad[4], wz = S.grad[5];
                const float th = sqrtf(wx * wx + wy * wy + wz * wz);
                float sh, ch, nq4[4];
                sincosf(0.5f * th, &sh, &ch);
                const float k = th > 1e-12f ? sh / th : 0.5f;
                rotate_quat(ch, k * wx, k * wy, k * wz, S.best + 3, nq4);
                S.geno[3] = nq4[0]; S.geno[4] = nq4[1]; S.geno[5] = nq4[2]; S.geno[6] = nq4[3];
            }
            __syncwarp();
            float ei, ea;
            e = __shfl_sync(kFull, eval_pose<false>(L, G, P, S, lane, ei, ea), 0);
            ++evals;
            ok = e < E;
            if (ok) {
#pragma unroll
                for (int c = 0; c < 3; ++c) bias[c] = P.sw_bias_keep * bias[c] + P.sw_bias_gain * (sg * delta[c]);
            }
        }
        if (ok) {
            for (int d = lane; d < Gn; d += 32) S.best[d] = S.geno[d];
            E = e; ++ns; nf = 0;
        } else {
#pragma unroll
            for (int c = 0; c < 3; ++c) bias[c] *= P.sw_bias_decay;
            ++nf; ns = 0;
        }
        __syncwarp();
        if (ns >= P.sw_max_succ) { rho *= P.sw_expand; ns = 0; }
        else if (nf >= P.sw_max_fail) { rho *= P.sw_contract; nf = 0; }
        if (trace && lane == 0) trace[it] = E;
        ++it;
    }
    return E;
}

}  // namespace adock
