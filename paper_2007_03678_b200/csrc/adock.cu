// adock.cu -- C-ABI entry points (include/adock.h) and the CUDA kernels behind them.
// Every step of the hot path runs in the kernels of this file / device.cuh; the host code only
// validates arguments, preprocesses the ligand topology once (topology.hpp) and launches.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <atomic>
#include <chrono>
#include <numeric>
#include <string>
#include <thread>
#include <vector>

#include "../../include/adock.h"
#include "device.cuh"
#include "lane.cuh"

using namespace adock;

// =================================================================== handles and errors
struct adock_grids {
    GridDev dev{};
    int M = 0;
    float4* cells = nullptr;
};

struct adock_ligand {
    Topology tp;
    unsigned char* d_blob = nullptr;
    int* d_ext_of_int = nullptr;
    int blob_bytes = 0;
    int scratch_floats = 0;
    float w_desolv = 0, qasp = 0, elec_scale = 0;
    double elec_fold = 1;                   // lane_elec_fold of the parameters the lane image was built with
    LaneImage lane;                         // image of the lane-per-individual kernels (lane_image.hpp)
    unsigned char* d_lane = nullptr;
    int lane_bytes = 0, lane_npad = 0, lane_own = 0;      // group scratch = lane_group_floats(npad, own, R, K) per lane
    bool owns_dev = true;                   // false: the device images live in a batch slab of adock_screen
};

static thread_local std::string g_err;
static thread_local long long g_launches = 0;
static int g_path = 0;                                    // adock_set_path: 0 auto, 1 warp per individual, 2 lane per individual
static int g_lane_var = -1;                               // lane-kernel variant forced by adock_set_path(21|22|24|41|42|43); -1 = by size
static thread_local bool g_prof = false;                  // adock_profile: time every dock_ls_kernel launch
static thread_local double g_ls_ms = 0;
static thread_local long long g_ls_launches = 0, g_ls_evals = 0;
static thread_local int g_last_dock_path = 0;             // kernel family of the last docking's local search

static int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
#define CUDA_TRY(expr)                                                                     \
    do {                                                                                   \
        cudaError_t e_ = (expr);                                                           \
        if (e_ != cudaSuccess) return fail(ADOCK_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
    } while (0)

extern "C" const char* adock_last_error(void) { return g_err.c_str(); }
extern "C" long long adock_launch_count(int reset) {
    long long v = g_launches;
    if (reset) g_launches = 0;
    return v;
}

extern "C" int adock_profile(int enable) {
    g_prof = enable != 0;
    g_ls_ms = 0; g_ls_launches = 0; g_ls_evals = 0;
    return ADOCK_OK;
}
extern "C" int adock_profile_read(double* ls_ms, long long* ls_launches, long long* ls_evals) {
    if (ls_ms) *ls_ms = g_ls_ms;
    if (ls_launches) *ls_launches = g_ls_launches;
    if (ls_evals) *ls_evals = g_ls_evals;
    return ADOCK_OK;
}

extern "C" int adock_default_params(adock_params* p) {
    if (!p) return fail(ADOCK_EINVAL, "params is NULL");
    p->elec_scale = (float)(0.1406 * 332.06363);
    p->diel_A = -8.5525f; p->diel_B = 86.9525f; p->diel_k = 7.7839f; p->diel_lambda = 0.003627f;
    p->w_desolv = 0.1322f; p->ds_sigma = 3.6f; p->qasp = 0.01097f; p->r_min = 0.5f; p->k_wall = 1000.0f;
    p->ad_rho = 0.8f; p->ad_eps = 1e-2f; p->lsrat = 0.06f;
    p->tourn_prob = 0.60f; p->xover_rate = 0.80f; p->mut_rate = 0.02f; p->dmov = 2.0f; p->dang = 1.57079632679489662f;
    p->lsit = 300; p->max_gens = 27000;
    p->ls_method = 0; p->sw_max_succ = 4; p->sw_max_fail = 4; p->autostop = 0; p->as_window = 10;
    p->sw_rho0 = 1.0f; p->sw_rho_lb = 0.01f; p->sw_expand = 2.0f; p->sw_contract = 0.5f;
    p->sw_bias_keep = 0.6f; p->sw_bias_gain = 0.4f; p->sw_bias_decay = 0.5f; p->as_tol = 0.15f;
    return ADOCK_OK;
}

// the lane image's electrostatic row coefficients are elec_scale q_i q_j / s with s = B lambda B (1 for a constant dielectric)
static double lane_elec_fold(const adock_params& p) {
    const double s = (double)p.diel_B * (double)p.diel_lambda * (double)p.diel_B;
    return s != 0.0 ? s : 1.0;
}
static ParDev make_pardev(const adock_params& p) {
    const double log2e = 1.4426950408889634;
    ParDev d;
    d.elec_sqrt = (float)std::sqrt((double)p.elec_scale); d.diel_A = p.diel_A; d.diel_B = p.diel_B; d.diel_k = p.diel_k;
    d.BlamB = (float)((double)p.diel_B * (double)p.diel_lambda * (double)p.diel_B);
    d.mlamB_log2e = (float)(-(double)p.diel_lambda * (double)p.diel_B * log2e);
    d.log2_dk = (float)std::log2((double)p.diel_k);
    {   // lane kernels (lane.cuh, pair_row): constants of eps(r) scaled by s = B lambda B; a constant dielectric (s = 0) is
        // passed as A = eps, B = 0, k exp(..) = 0 with s = 1
        const double s = lane_elec_fold(p);
        if ((double)p.diel_B * (double)p.diel_lambda * (double)p.diel_B != 0.0) { d.diel_As = (float)((double)p.diel_A / s); d.diel_Bs = (float)((double)p.diel_B / s); }
        else { d.diel_As = (float)((double)p.diel_A + (double)p.diel_B / (1.0 + (double)p.diel_k)); d.diel_Bs = 0.f; d.log2_dk = -INFINITY; d.mlamB_log2e = 0.f; }
    }
    d.inv_sig2 = (float)(1.0 / ((double)p.ds_sigma * (double)p.ds_sigma));
    d.mhalf_inv_sig2_log2e = (float)(-0.5 * log2e / ((double)p.ds_sigma * (double)p.ds_sigma));
    d.rmin2 = p.r_min * p.r_min; d.k_wall = p.k_wall; d.k_wall_h = 0.f;    // k_wall_h set per grid
    d.ad_rho = p.ad_rho; d.ad_eps = p.ad_eps;
    d.tourn_prob = p.tourn_prob; d.xover_rate = p.xover_rate; d.mut_rate = p.mut_rate; d.dmov = p.dmov; d.dang = p.dang;
    d.lsit = p.lsit;
    d.ls_method = p.ls_method; d.sw_max_succ = p.sw_max_succ; d.sw_max_fail = p.sw_max_fail;
    d.autostop = p.autostop; d.as_window = p.as_window;
    d.sw_rho0 = p.sw_rho0; d.sw_rho_lb = p.sw_rho_lb; d.sw_expand = p.sw_expand; d.sw_contract = p.sw_contract;
    d.sw_bias_keep = p.sw_bias_keep; d.sw_bias_gain = p.sw_bias_gain; d.sw_bias_decay = p.sw_bias_decay; d.as_tol = p.as_tol;
    return d;
}

static int check_params(const adock_params* in, const adock_ligand* l, adock_params& out) {
    if (in) out = *in; else adock_default_params(&out);
    const float* f = &out.elec_scale;
    for (int i = 0; i < 18; ++i)
        if (!std::isfinite(f[i])) return fail(ADOCK_EINVAL, "non-finite parameter");
    if (!(out.ds_sigma > 0) || !(out.r_min > 0) || !(out.elec_scale >= 0) || out.lsit < 0 || out.max_gens < 0 || !(out.ad_eps > 0) ||
        !(out.diel_k > 0))      // k <= 0 puts a pole into eps(r); the kernels evaluate k exp(-lambda B r) as 2^(.. + log2 k)
        return fail(ADOCK_EINVAL, "parameter out of range");
    const float* f2 = &out.sw_rho0;
    for (int i = 0; i < 7; ++i)
        if (!std::isfinite(f2[i])) return fail(ADOCK_EINVAL, "non-finite parameter");
    if (out.ls_method < 0 || out.ls_method > 1 || out.sw_max_succ < 1 || out.sw_max_fail < 1 || !(out.sw_rho0 > 0) ||
        !(out.sw_expand > 0) || !(out.sw_contract > 0) || std::isnan(out.as_tol) || (out.autostop && (out.as_window < 1 || out.as_window > kAsMaxWindow)))
        return fail(ADOCK_EINVAL, "parameter out of range");
    if (l && !l->d_blob) return fail(ADOCK_EINVAL, "host-only ligand handle (loaded with grids == NULL)");
    if (l && (out.w_desolv != l->w_desolv || out.qasp != l->qasp || out.elec_scale != l->elec_scale || lane_elec_fold(out) != l->elec_fold))
        return fail(ADOCK_EINVAL, "elec_scale/w_desolv/qasp/diel_B/diel_lambda differ from the values baked into the ligand at load time");
    return ADOCK_OK;
}

// =================================================================== grids
// caller's [M][nz][ny][nx] maps -> xy-patch cells per (type, charge sign): cells[2t + s][z][y][x] (y < ny-1, x < nx-1)
// = one 32-byte sector {a_t, pm}(x,y) {a_t, pm}(x+1,y) | {a_t, pm}(x,y+1) {a_t, pm}(x+1,y+1) of plane z, with
// pm = elec + desolv (s = 0) or elec - desolv (s = 1)   (device.cuh, grid term)
__global__ void relayout_kernel(const float* __restrict__ maps, float4* __restrict__ cells, int T, int nx, int ny, int nz) {
    const long long per_set = (long long)nz * (ny - 1) * (nx - 1);
    const long long ncell = 2ll * T * per_set;
    const long long plane = (long long)nz * ny * nx;
    const float* el = maps + T * plane;
    const float* ds = maps + (T + 1) * plane;
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(c % (nx - 1));
        const long long row = c / (nx - 1);               // (set*nz + z)*(ny-1) + y
        const int iy = (int)(row % (ny - 1));
        const long long sz = row / (ny - 1);               // set*nz + z
        const int iz = (int)(sz % nz), set = (int)(sz / nz);
        const float* at = maps + (set >> 1) * plane;
        const float sg = (set & 1) ? -1.f : 1.f;
        const long long p = ((long long)iz * ny + iy) * nx + ix, p1 = p + nx;
        cells[2 * c] = make_float4(at[p], el[p] + sg * ds[p], at[p + 1], el[p + 1] + sg * ds[p + 1]);
        cells[2 * c + 1] = make_float4(at[p1], el[p1] + sg * ds[p1], at[p1 + 1], el[p1 + 1] + sg * ds[p1 + 1]);
    }
}

extern "C" int adock_load_grids(const float* host_maps, int M, int nx, int ny, int nz, float spacing, const float origin[3],
                                adock_grids** out) {
    if (!host_maps || !origin || !out) return fail(ADOCK_EINVAL, "NULL argument");
    if (M < 3 || nx < 2 || ny < 2 || nz < 2 || !(spacing > 0) || !std::isfinite(spacing)) return fail(ADOCK_EINVAL, "bad grid shape");
    if (M > ADOCK_MAX_MAPS) return fail(ADOCK_ELIMIT, "more than ADOCK_MAX_MAPS maps");
    if (nx > 1024 || ny > 1024 || nz > 1024) return fail(ADOCK_ELIMIT, "grid dimension above 1024");
    const size_t npts = (size_t)nx * ny * nz;
    for (size_t i = 0; i < (size_t)M * npts; ++i)
        if (!std::isfinite(host_maps[i])) return fail(ADOCK_EINVAL, "non-finite map value");
    const int T = M - 2;
    float* d_raw = nullptr;
    float4* cells = nullptr;
    const size_t ncell = (size_t)2 * T * nz * (ny - 1) * (nx - 1);
    cudaError_t e = cudaMalloc(&d_raw, (size_t)M * npts * sizeof(float));
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("cudaMalloc: ") + cudaGetErrorString(e));
    e = cudaMalloc(&cells, ncell * 2 * sizeof(float4));
    if (e != cudaSuccess) { cudaFree(d_raw); return fail(e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("cudaMalloc: ") + cudaGetErrorString(e)); }
    e = cudaMemcpy(d_raw, host_maps, (size_t)M * npts * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        relayout_kernel<<<1184, 256>>>(d_raw, cells, T, nx, ny, nz);
        ++g_launches;
        e = cudaDeviceSynchronize();
    }
    cudaFree(d_raw);
    if (e != cudaSuccess) { cudaFree(cells); return fail(ADOCK_ECUDA, std::string("grid upload: ") + cudaGetErrorString(e)); }
    adock_grids* g = new adock_grids;
    g->M = M; g->cells = cells;
    g->dev.cells = cells;
    g->dev.set_stride = (long long)nz * (ny - 1) * (nx - 1) * 2;
    g->dev.nx = nx; g->dev.ny = ny; g->dev.nz = nz; g->dev.T = T;
    g->dev.h = spacing; g->dev.inv_h = 1.0f / spacing;
    g->dev.ox = origin[0]; g->dev.oy = origin[1]; g->dev.oz = origin[2];
    g->dev.bx = spacing * (nx - 1); g->dev.by = spacing * (ny - 1); g->dev.bz = spacing * (nz - 1);
    *out = g;
    return ADOCK_OK;
}

extern "C" void adock_free_grids(adock_grids* g) {
    if (!g) return;
    cudaFree(g->cells);
    delete g;
}

// =================================================================== ligand
extern "C" int adock_load_ligand(const adock_grids* grids, const adock_params* params, int N, const float* xyz, const int* type,
                                 const float* charge, int nbonds, const int* bonds, int R, const int* rot_bonds, int root_atom,
                                 int T, const float* pair_coeffs, const float* solpar, const float* vol, adock_ligand** out) {
    if (!xyz || !type || !charge || !pair_coeffs || !solpar || !vol || !out || (nbonds > 0 && !bonds) || (R > 0 && !rot_bonds))
        return fail(ADOCK_EINVAL, "NULL argument");
    if (N < 1 || R < 0 || T < 1 || nbonds < 0 || root_atom < 0 || root_atom >= N) return fail(ADOCK_EINVAL, "bad ligand shape");
    if (N > ADOCK_MAX_ATOMS || R > ADOCK_MAX_TORSIONS) return fail(ADOCK_ELIMIT, "ligand exceeds ADOCK_MAX_ATOMS / ADOCK_MAX_TORSIONS");
    if (grids && T + 2 > grids->M) return fail(ADOCK_EINVAL, "ligand atom types exceed the loaded maps");
    adock_params p;
    int rc = check_params(params, nullptr, p);
    if (rc) return rc;
    for (int i = 0; i < N; ++i) {
        if (type[i] < 0 || type[i] >= T) return fail(ADOCK_EINVAL, "atom type out of range");
        if (!std::isfinite(charge[i]) || !std::isfinite(xyz[3 * i]) || !std::isfinite(xyz[3 * i + 1]) || !std::isfinite(xyz[3 * i + 2]))
            return fail(ADOCK_EINVAL, "non-finite ligand input");
    }
    for (int i = 0; i < T * T * 4; ++i) if (!std::isfinite(pair_coeffs[i])) return fail(ADOCK_EINVAL, "non-finite pair coefficient");
    for (int i = 0; i < T * T; ++i)         // the kernels evaluate r^-6 and r^-10 only (R5)
        if (pair_coeffs[4 * i + 2] != 6.0f && pair_coeffs[4 * i + 2] != 10.0f) return fail(ADOCK_EINVAL, "pair exponent expA must be 6 or 10");
    for (int i = 0; i < T; ++i) if (!std::isfinite(solpar[i]) || !std::isfinite(vol[i])) return fail(ADOCK_EINVAL, "non-finite solpar / vol");
    adock_ligand* l = new adock_ligand;
    if (!build_topology(l->tp, N, xyz, type, charge, nbonds, bonds, R, rot_bonds, root_atom, T, pair_coeffs, solpar, vol, p.w_desolv, p.qasp)) {
        std::string msg = l->tp.error;
        delete l;
        return fail(ADOCK_EINVAL, msg);
    }
    l->w_desolv = p.w_desolv; l->qasp = p.qasp; l->elec_scale = p.elec_scale; l->elec_fold = lane_elec_fold(p);
    build_lane_image(l->lane, l->tp, xyz, type, charge, pair_coeffs, solpar, vol, p.w_desolv, p.qasp, (double)p.elec_scale / l->elec_fold);
    l->lane_bytes = (int)l->lane.blob.size();
    l->lane_npad = l->lane.npad; l->lane_own = l->lane.own_floats;
    l->blob_bytes = (int)l->tp.blob.size();
    l->scratch_floats = warp_scratch_floats(N, l->tp.nfrag, R);
    if (16 + l->blob_bytes + 4 * l->scratch_floats > 227 * 1024) {
        delete l;
        return fail(ADOCK_ELIMIT, "ligand image does not fit in shared memory");
    }
    if (!grids) {           // host-only handle: integer structure and image for inspection
        *out = l;
        return ADOCK_OK;
    }
    cudaError_t e = cudaMalloc(&l->d_blob, l->blob_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&l->d_ext_of_int, l->tp.ext_of_int.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&l->d_lane, l->lane_bytes);
    if (e == cudaSuccess) e = cudaMemcpy(l->d_lane, l->lane.blob.data(), l->lane_bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(l->d_blob, l->tp.blob.data(), l->blob_bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(l->d_ext_of_int, l->tp.ext_of_int.data(), l->tp.ext_of_int.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(l->d_blob); cudaFree(l->d_ext_of_int); cudaFree(l->d_lane);
        delete l;
        return fail(e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("ligand upload: ") + cudaGetErrorString(e));
    }
    *out = l;
    return ADOCK_OK;
}

extern "C" void adock_free_ligand(adock_ligand* l) {
    if (!l) return;
    if (l->owns_dev) {
        cudaFree(l->d_blob);
        cudaFree(l->d_ext_of_int);
        cudaFree(l->d_lane);
    }
    delete l;
}

extern "C" int adock_ligand_pairs(const adock_ligand* l, int* npairs, const int** ij) {
    if (!l || !npairs || !ij) return fail(ADOCK_EINVAL, "NULL argument");
    *npairs = (int)l->tp.pairs.size() / 2;
    *ij = l->tp.pairs.data();
    return ADOCK_OK;
}

extern "C" int adock_ligand_tree(const adock_ligand* l, const int** tor_order, const unsigned char** moved, const int** rot,
                                 const float** pivot) {
    if (!l) return fail(ADOCK_EINVAL, "NULL argument");
    if (tor_order) *tor_order = l->tp.tor_order.data();
    if (moved) *moved = l->tp.moved.data();
    if (rot) *rot = l->tp.rot.data();
    if (pivot) *pivot = l->tp.pivot;
    return ADOCK_OK;
}

extern "C" int adock_ligand_image(const adock_ligand* l, int* bytes, const unsigned char** image, const int** int_of_ext) {
    if (!l || !bytes || !image) return fail(ADOCK_EINVAL, "NULL argument");
    *bytes = l->blob_bytes;
    *image = l->tp.blob.data();
    if (int_of_ext) *int_of_ext = l->tp.int_of_ext.data();
    return ADOCK_OK;
}

extern "C" int adock_ligand_lane_image(const adock_ligand* l, int* bytes, const unsigned char** image, const int** pos_of_ext) {
    if (!l || !bytes || !image) return fail(ADOCK_EINVAL, "NULL argument");
    *bytes = l->lane_bytes;
    *image = l->lane.blob.data();
    if (pos_of_ext) *pos_of_ext = l->lane.pos_of_ext.data();
    return ADOCK_OK;
}

extern "C" int adock_last_dock_path(void) { return g_last_dock_path; }

extern "C" int adock_set_path(int path) {
    if (path == 21 || path == 22 || path == 24) { g_path = 2; g_lane_var = path == 21 ? 0 : path == 22 ? 1 : 2; return ADOCK_OK; }
    if (path == 41 || path == 42 || path == 43) { g_path = 2; g_lane_var = path - 38; return ADOCK_OK; }
    if (path < 0 || path > 3)
        return fail(ADOCK_EINVAL, "path must be 0 (auto), 1 (warp per individual), 2 (lane per individual), 21/22/24 (1, 2, 4 warps per group, "
                                  "positions in shared memory), 41/42/43 (positions in tensor memory, 8/12/16 warps per SM) or 3 (team per individual)");
    g_path = path; g_lane_var = -1;
    return ADOCK_OK;
}

// =================================================================== launch geometry
static int g_sm_count = 0, g_smem_optin = 0;
static int device_props() {
    if (g_sm_count) return ADOCK_OK;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev));
    CUDA_TRY(cudaDeviceGetAttribute(&g_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    return ADOCK_OK;
}
static size_t cta_smem(int blob_bytes, int scratch_floats, int warps) { return 16 + (size_t)blob_bytes + (size_t)warps * scratch_floats * 4; }
// largest warp count <= want whose shared memory fits
static int fit_warps(int blob_bytes, int scratch_floats, int want) {
    int w = want;
    while (w > 1 && cta_smem(blob_bytes, scratch_floats, w) > (size_t)g_smem_optin) w >>= 1;
    return cta_smem(blob_bytes, scratch_floats, w) <= (size_t)g_smem_optin ? w : 0;
}

// =================================================================== scoring kernel (rows a1-a4)
struct ScoreArgs {
    const unsigned char* blob;
    const float* genos;
    float* E;
    float* terms;
    float* grads;
    int blob_bytes, n, gstride, dstride;
};

template <bool GRAD>
__global__ void __launch_bounds__(256) score_kernel(GridDev G, ParDev P, ScoreArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* blob = smem + 16;
    stage_ligand(blob, a.blob, a.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);
    const LigS L = lig_view(blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const WarpS S = warp_view(reinterpret_cast<float*>(blob + a.blob_bytes) + (size_t)warp * warp_scratch_floats(L.N, L.nfrag, L.R), L);
    const int Gn = 7 + L.R, D = 6 + L.R;
    for (int idx = blockIdx.x * W + warp; idx < a.n; idx += gridDim.x * W) {
        for (int d = lane; d < Gn; d += 32) S.geno[d] = a.genos[(size_t)idx * a.gstride + d];
        __syncwarp();
        float ei, ea;
        const float e = eval_pose<GRAD>(L, G, P, S, lane, ei, ea);
        if (lane == 0) {
            a.E[idx] = e;
            if (a.terms) { a.terms[2 * (size_t)idx] = ei; a.terms[2 * (size_t)idx + 1] = ea; }
        }
        if (GRAD)
            for (int d = lane; d < D; d += 32) a.grads[(size_t)idx * a.dstride + d] = S.grad[d];
        __syncwarp();
    }
}


// =================================================================== lane-per-individual geometry (lane.cuh)
// A group of K warps shares 32 individuals.  A variant of the lane kernels fixes K, the most warps per CTA W (the register
// budget is 64 K / (32 W) per thread: 255 at 8 warps, 168 at 12, 128 at 16) and where the atom positions live: shared
// memory, or tensor memory (TM; one warp per group only), which takes 62 % of the per-lane state of a 40-atom ligand out
// of shared memory so that 12 or 16 warps fit where 8 did.
template <int K_, int W_, bool TM_> struct LaneCfg {
    static constexpr int K = K_, kMaxWarps = W_;
    static constexpr bool TM = TM_;
    static constexpr bool ST = TM_;         // local-search state in shared memory (the room the positions left) instead of global columns
};
struct LaneVar { int K, W; bool TM; double eff, eff_ls; };   // measured throughput per SM at full residency (K = 1 with 8 warps = 1):
                                                              // eff of the scoring kernels, eff_ls of the local-search kernels
constexpr int kNumLaneVars = 6;
// profiles/r02_lane_variants.md (sweep40 / drug).  16 warps leave the local-search kernels 128 registers (spills) and no room
// for the chain state in shared memory.
static const LaneVar kLaneVars[kNumLaneVars] = {{1, 8, false, 1.0, 1.0},  {2, 12, false, 1.04, 1.0}, {4, 16, false, 0.90, 0.78},
                                                {1, 8, true, 1.02, 0.97}, {1, 12, true, 1.18, 1.21}, {1, 16, true, 1.23, 0.70}};
#define LANE_VARIANT(v, ...)                                                      \
    switch (v) {                                                                  \
        case 0: { using C = LaneCfg<1, 8, false>; __VA_ARGS__; } break;           \
        case 1: { using C = LaneCfg<2, 12, false>; __VA_ARGS__; } break;          \
        case 2: { using C = LaneCfg<4, 16, false>; __VA_ARGS__; } break;          \
        case 3: { using C = LaneCfg<1, 8, true>; __VA_ARGS__; } break;            \
        case 4: { using C = LaneCfg<1, 12, true>; __VA_ARGS__; } break;           \
        default: { using C = LaneCfg<1, 16, true>; __VA_ARGS__; } break;          \
    }
struct LaneGeom { int bytes, npad, own, R; };            // of the largest ligand of a launch
static LaneGeom lane_geom(const adock_ligand* l) { return LaneGeom{l->lane_bytes, l->lane_npad, l->lane_own, l->tp.R}; }
static LaneGeom lane_geom_max(LaneGeom a, LaneGeom b) {
    return LaneGeom{std::max(a.bytes, b.bytes), std::max(a.npad, b.npad), std::max(a.own, b.own), std::max(a.R, b.R)};
}
// ls: a local-search kernel (the TM variants keep the chain state in shared memory)
static int lane_var_floats(const LaneGeom& g, int v, bool ls) {
    return lane_group_floats(g.npad, g.own, g.R, kLaneVars[v].K, kLaneVars[v].TM, ls && kLaneVars[v].TM);
}
// shared memory of a CTA of `groups` groups with `nimg` image slots
static size_t lane_smem(const LaneGeom& g, int v, bool ls, int groups, int nimg = 1) {
    const size_t slot = ((size_t)g.bytes + 127) & ~(size_t)127;
    return 16 + (size_t)nimg * slot + (size_t)groups * lane_var_floats(g, v, ls) * 128;
}
static bool lane_fits(const LaneGeom& g, int v, bool ls, int groups, int nimg = 1) {
    if (kLaneVars[v].TM && 3 * g.npad > lane_tmem_columns(groups * kLaneVars[v].K)) return false;
    return lane_smem(g, v, ls, groups, nimg) <= (size_t)g_smem_optin;
}
// most groups per CTA that fit (0: not even one)
static int lane_fit_groups(const LaneGeom& g, int v, bool ls) {
    int n = kLaneVars[v].W / kLaneVars[v].K;
    while (n > 0 && !lane_fits(g, v, ls, n)) --n;
    return n;
}
// the lane kernels want at least one warp per scheduler
static bool lane_ok(const adock_ligand* l) {
    const LaneGeom g = lane_geom(l);
    for (int v = 0; v < kNumLaneVars; ++v)
        if (lane_fit_groups(g, v, true) * kLaneVars[v].K >= 4) return true;
    return false;
}
// ADADELTA chains (threads) from which the lane-per-individual kernels are preferred over warp-per-individual
static long long lane_min_chains() { return (long long)g_sm_count * 42; }     // measured cross-over on the drug config: 34 ligands x 180 chains (the lane kernel's partial wave costs the same from 1 to 64 ligands)
// ---- launch plan of a lane-per-individual kernel over `total` groups of 32 individuals, `jg` consecutive groups per
// ligand image (jg >= total: one image).  CTA b takes groups [b*ng, (b+1)*ng) and stages every image they touch.
struct LanePlan {
    int var = -1;           // variant (-1: nothing fits)
    int K = 0;              // its warps per group
    int ng = 0;             // groups per CTA
    int nctas = 0;
    int nimg = 1;           // image slots per CTA
    int slot = 0;           // bytes per image slot (multiple of 128)
    int gfloats = 0;        // floats per lane between groups
    size_t smem = 0;
};
static int lane_plan_images(long long total, int jg, int ng) {        // most images any CTA of the partition touches
    if (jg >= total) return 1;
    int worst = 1;
    for (long long first = 0; first < total; first += ng) {
        const long long last = std::min<long long>(first + ng, total) - 1;
        worst = std::max(worst, (int)(last / jg - first / jg) + 1);
        if (worst >= (ng - 1) / jg + 2) break;                          // the bound is reached
    }
    return worst;
}
// Model: an SM with w resident warps of a variant works at min(w, W)/W of the variant's rate eff (measured per SM at
// full residency: profiles/r02_lane_variants.md); waves of CTAs run one after another.
static LanePlan lane_plan(const LaneGeom& g, long long total, int jg, bool ls) {
    LanePlan best;
    double best_t = 1e300;
    if (total < 1) total = 1;
    if (jg < 1) jg = 1;
    for (int v = 0; v < kNumLaneVars; ++v) {
        if (g_lane_var >= 0 && v != g_lane_var) continue;       // a forced variant that does not fit is an error (ADOCK_ELIMIT), never a silent substitute
        const LaneVar& V = kLaneVars[v];
        for (int ng = V.W / V.K; ng >= 1; --ng) {
            if (!lane_fits(g, v, ls, ng, lane_plan_images(total, jg, ng))) continue;
            const long long nctas = (total + ng - 1) / ng, waves = (nctas + g_sm_count - 1) / g_sm_count;
            const double t = (double)waves * ng / ((ls ? V.eff_ls : V.eff) * (double)(ng * V.K) / V.W);
            if (t < best_t * 0.999) {
                best_t = t;
                best.var = v; best.ng = ng;
            }
        }
    }
    if (best.var < 0) return best;
    best.K = kLaneVars[best.var].K;
    best.nctas = (int)((total + best.ng - 1) / best.ng);
    best.nimg = lane_plan_images(total, jg, best.ng);
    best.slot = (g.bytes + 127) & ~127;
    best.gfloats = lane_var_floats(g, best.var, ls);
    best.smem = lane_smem(g, best.var, ls, best.ng, best.nimg);
    return best;
}
// variant for `ngroups` groups of 32 individuals of one ligand (-1: none fits)
static int lane_pick_var(const LaneGeom& g, long long ngroups, bool ls) { return lane_plan(g, ngroups, (int)std::min<long long>(ngroups, 1 << 30), ls).var; }
// groups per CTA of a launch of `ngroups` groups on one CTA per SM (each looping over its share, or wave after wave):
// passes x time of a pass, where an SM with w = n K resident warps works at w / (w + 4) of its full rate (fitted to the
// measured variants: 8 / 12 / 16 warps = 0.83 / 0.94 / 1 of the 16-warp rate), i.e. a pass of n groups lasts ~ n K + 4
static int lane_spread_groups(int fit, long long ngroups, int K) {
    int best = fit;
    long long best_cost = -1;
    for (int n = fit; n >= 1; --n) {
        const long long passes = (ngroups + (long long)g_sm_count * n - 1) / ((long long)g_sm_count * n);
        const long long cost = passes * (n * K + 4);
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = n; }
    }
    return best;
}

template <bool GRAD, class C>
__global__ void __launch_bounds__(C::kMaxWarps * 32, 1) score_lane_kernel(GridDev G, ParDev P, ScoreArgs a) {
    constexpr int K = C::K;
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* blob = smem + 16;
    stage_ligand(blob, a.blob, a.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);
    const uint32_t tmem = lane_tmem_open<C::TM>(smem);
    const LaneL L = lane_view(blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NG = (blockDim.x >> 5) / K;
    const LaneS S = lane_scratch<K, C::TM>(reinterpret_cast<float*>(blob + a.blob_bytes), L, warp, lane, 0, tmem);
    const int Gn = 7 + L.R;
    const int nchunks = (a.n + 31) >> 5;
    for (int c = blockIdx.x * NG + S.gid; c < nchunks; c += gridDim.x * NG) {
        const int idx = c * 32 + lane;
        const bool act = idx < a.n;
        const int src = act ? idx : a.n - 1;
        if (S.part == 0)
            for (int d = 0; d < Gn; ++d) S.geno[d * 32] = a.genos[(size_t)src * a.gstride + d];
        group_sync<K>(S);
        float ei, ea;
        bool gf;
        const float e = lane_eval<GRAD, K, 1, C::TM, C::kMaxWarps == 16>(L, G, P, S, GRAD ? a.grads + (size_t)src * a.dstride : nullptr, 1, act, ei, ea, gf);
        if (act && S.part == 0) {
            a.E[idx] = e;
            if (a.terms) { a.terms[2 * (size_t)idx] = ei; a.terms[2 * (size_t)idx + 1] = ea; }
        }
        group_sync<K>(S);                               // part 0 is done with the positions and own[]
    }
    lane_tmem_close<C::TM>(tmem);
}

template <bool GRAD, class C>
static int launch_score_lane_k(const adock_grids* grids, const adock_ligand* lig, const ParDev& P, const ScoreArgs& a, int var, int ngroups,
                               cudaStream_t st) {
    const LaneGeom g = lane_geom(lig);
    const int NG = lane_spread_groups(lane_fit_groups(g, var, false), ngroups, C::K);
    const size_t smem = lane_smem(g, var, false, NG);
    const int grid = (int)std::max<long long>(1, std::min<long long>(((long long)ngroups + NG - 1) / NG, g_sm_count));
    CUDA_TRY(cudaFuncSetAttribute(score_lane_kernel<GRAD, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    score_lane_kernel<GRAD, C><<<grid, NG * C::K * 32, smem, st>>>(grids->dev, P, a);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return ADOCK_OK;
}

static int launch_score_lane(const adock_grids* grids, const adock_ligand* lig, const adock_params& p, const float* d_genos, int n,
                             int gstride, float* d_E, float* d_terms, float* d_grads, int dstride, cudaStream_t st) {
    const int ngroups = (n + 31) / 32;
    const int var = lane_pick_var(lane_geom(lig), ngroups, false);
    if (var < 0) return fail(ADOCK_ELIMIT, "ligand does not fit the lane-per-individual kernel");
    ParDev P = make_pardev(p);
    P.k_wall_h = p.k_wall * grids->dev.h;
    ScoreArgs a{lig->d_lane, d_genos, d_E, d_terms, d_grads, lig->lane_bytes, n, gstride, dstride};
    int rc = ADOCK_OK;
    if (d_grads) { LANE_VARIANT(var, rc = launch_score_lane_k<true, C>(grids, lig, P, a, var, ngroups, st)) }
    else { LANE_VARIANT(var, rc = launch_score_lane_k<false, C>(grids, lig, P, a, var, ngroups, st)) }
    return rc;
}

static int launch_score(const adock_grids* grids, const adock_ligand* lig, const adock_params& p, const float* d_genos, int n,
                        int gstride, float* d_E, float* d_terms, float* d_grads, int dstride, cudaStream_t st) {
    int rc = device_props();
    if (rc) return rc;
    if (g_path == 2 || (g_path == 0 && n >= 2048 && lane_ok(lig)))
        return launch_score_lane(grids, lig, p, d_genos, n, gstride, d_E, d_terms, d_grads, dstride, st);
    const int W = fit_warps(lig->blob_bytes, lig->scratch_floats, 8);
    if (!W) return fail(ADOCK_ELIMIT, "ligand does not fit in shared memory");
    const size_t smem = cta_smem(lig->blob_bytes, lig->scratch_floats, W);
    ParDev P = make_pardev(p);
    P.k_wall_h = p.k_wall * grids->dev.h;
    ScoreArgs a{lig->d_blob, d_genos, d_E, d_terms, d_grads, lig->blob_bytes, n, gstride, dstride};
    int per_sm = 1;
    if (d_grads) {
        CUDA_TRY(cudaFuncSetAttribute(score_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, score_kernel<true>, W * 32, smem));
    } else {
        CUDA_TRY(cudaFuncSetAttribute(score_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, score_kernel<false>, W * 32, smem));
    }
    if (per_sm < 1) per_sm = 1;
    long long want = ((long long)n + W - 1) / W;
    int grid = (int)std::min<long long>(want, (long long)g_sm_count * per_sm);       // persistent: a multiple of the SM count
    if (grid < 1) grid = 1;
    if (d_grads) score_kernel<true><<<grid, W * 32, smem, st>>>(grids->dev, P, a);
    else score_kernel<false><<<grid, W * 32, smem, st>>>(grids->dev, P, a);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return ADOCK_OK;
}

extern "C" int adock_score_batch(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                                 const float* d_genotypes, int n, int gstride, float* d_energies, float* d_energy_terms,
                                 float* d_gradients, int dstride, void* cuda_stream) {
    if (!grids || !ligand) return fail(ADOCK_EINVAL, "NULL handle");
    if (n < 0) return fail(ADOCK_EINVAL, "n < 0");
    if (n == 0) return ADOCK_OK;
    if (!d_genotypes || !d_energies) return fail(ADOCK_EINVAL, "NULL buffer");
    if (gstride < 7 + ligand->tp.R || (d_gradients && dstride < 6 + ligand->tp.R)) return fail(ADOCK_EINVAL, "stride too small");
    adock_params p;
    int rc = check_params(params, ligand, p);
    if (rc) return rc;
    return launch_score(grids, ligand, p, d_genotypes, n, gstride, d_energies, d_energy_terms, d_gradients, dstride, (cudaStream_t)cuda_stream);
}

extern "C" int adock_score_batch_host(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                                      const float* h_genotypes, int n, int gstride, float* h_energies, float* h_energy_terms,
                                      float* h_gradients, int dstride, void* cuda_stream) {
    if (!grids || !ligand) return fail(ADOCK_EINVAL, "NULL handle");
    if (n < 0) return fail(ADOCK_EINVAL, "n < 0");
    if (n == 0) return ADOCK_OK;
    if (!h_genotypes || !h_energies) return fail(ADOCK_EINVAL, "NULL buffer");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float *dg = nullptr, *dE = nullptr, *dT = nullptr, *dG = nullptr;
    const size_t gb = (size_t)n * gstride * 4, db = (size_t)n * dstride * 4;
    CUDA_TRY(cudaMalloc(&dg, gb));
    int rc = ADOCK_OK;
    cudaError_t e = cudaMalloc(&dE, (size_t)n * 4);
    if (e == cudaSuccess && h_energy_terms) e = cudaMalloc(&dT, (size_t)n * 8);
    if (e == cudaSuccess && h_gradients) e = cudaMalloc(&dG, db);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dg, h_genotypes, gb, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) rc = adock_score_batch(grids, ligand, params, dg, n, gstride, dE, dT, dG, dstride, st);
    if (e == cudaSuccess && rc == ADOCK_OK) e = cudaMemcpyAsync(h_energies, dE, (size_t)n * 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && rc == ADOCK_OK && dT) e = cudaMemcpyAsync(h_energy_terms, dT, (size_t)n * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && rc == ADOCK_OK && dG) e = cudaMemcpyAsync(h_gradients, dG, db, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(dg); cudaFree(dE); cudaFree(dT); cudaFree(dG);
    if (e != cudaSuccess) return fail(ADOCK_ECUDA, std::string("score_batch_host: ") + cudaGetErrorString(e));
    return rc;
}

// =================================================================== Philox test hook (R8)
__global__ void philox_kernel(uint32_t k0, uint32_t k1, const uint4* ctr, int n, uint4* out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = philox4x32_10(k0, k1, ctr[i]);
}
extern "C" int adock_philox(const unsigned int key[2], const unsigned int* d_ctr, int n, unsigned int* d_out, void* cuda_stream) {
    if (!key || (n > 0 && (!d_ctr || !d_out)) || n < 0) return fail(ADOCK_EINVAL, "bad argument");
    if (n == 0) return ADOCK_OK;
    philox_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(key[0], key[1], (const uint4*)d_ctr, n, (uint4*)d_out);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return ADOCK_OK;
}

// =================================================================== local search on an array (row a5)
struct LsArgs {
    const unsigned char* blob;
    float* genos;
    float* E;
    int* iters;
    float* trace;
    int blob_bytes, n, gstride;
    unsigned long long seed;    // Solis-Wets (R11): Philox key; chain i draws with id = i, generation = gen
    unsigned int gen;
};

__global__ void __launch_bounds__(128) ls_array_kernel(GridDev G, ParDev P, LsArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* blob = smem + 16;
    stage_ligand(blob, a.blob, a.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);
    const LigS L = lig_view(blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const WarpS S = warp_view(reinterpret_cast<float*>(blob + a.blob_bytes) + (size_t)warp * warp_scratch_floats(L.N, L.nfrag, L.R), L);
    const int Gn = 7 + L.R;
    const int idx = blockIdx.x * W + warp;
    if (idx >= a.n) return;
    for (int d = lane; d < Gn; d += 32) S.geno[d] = a.genos[(size_t)idx * a.gstride + d];
    __syncwarp();
    int iters = 0;
    float* tr = a.trace ? a.trace + (size_t)idx * P.lsit : nullptr;
    const float e = P.ls_method == 1 ? solis_wets_search(L, G, P, S, lane, a.E[idx], a.seed, (uint32_t)idx, a.gen, iters, tr)
                                     : adadelta_search(L, G, P, S, lane, __int_as_float(0x7fc00000), iters, tr);
    for (int d = lane; d < Gn; d += 32) a.genos[(size_t)idx * a.gstride + d] = S.best[d];
    if (lane == 0) {
        a.E[idx] = e;
        if (a.iters) a.iters[idx] = iters;
    }
}

// team-per-chain variant (ADADELTA; the docking's dock_ls_team_kernel<TPC> on an array of starts): TPC teams of kTeamW warps per
// CTA, one chain each, sharing the ligand image
template <int TPC>
__global__ void __launch_bounds__(TPC * kTeamW * 32, TPC == 1 ? 5 : 1) ls_array_team_kernel(GridDev G, ParDev P, LsArgs a, int team_floats) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* blob = smem + 16;
    stage_ligand(blob, a.blob, a.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);
    const LigS L = lig_view(blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, team = warp / kTeamW;
    TeamS T = team_view(reinterpret_cast<float*>(blob + a.blob_bytes) + (size_t)team * team_floats, L, warp % kTeamW);
    T.bar = 1 + team;
    const int Gn = 7 + L.R;
    const size_t idx = (size_t)blockIdx.x * TPC + team;
    if (idx >= (size_t)a.n) return;                     // whole teams leave: the barriers below are per team
    if (T.wi == 0) for (int d = lane; d < Gn; d += 32) T.S.geno[d] = a.genos[idx * a.gstride + d];
    team_sync(T);
    int iters = 0;
    const float e = adadelta_search_team<TPC == 1 ? 2 : 4, TPC == 4>(L, G, P, T, lane, __int_as_float(0x7fc00000), iters,
                                                                     a.trace ? a.trace + idx * P.lsit : nullptr);
    if (T.wi == 0) {
        for (int d = lane; d < Gn; d += 32) a.genos[idx * a.gstride + d] = T.S.best[d];
        if (lane == 0) {
            a.E[idx] = e;
            if (a.iters) a.iters[idx] = iters;
        }
    }
}

// lane-per-individual variant: lane c of the launch's groups runs chain c; ADADELTA state in global scratch columns
// [row][all group lanes of the launch]
template <class C, bool SW>
__global__ void __launch_bounds__(C::kMaxWarps * 32, 1) ls_array_lane_kernel(GridDev G, ParDev P, LsArgs a, float* __restrict__ scratch) {
    constexpr int K = C::K;
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* blob = smem + 16;
    stage_ligand(blob, a.blob, a.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);
    const uint32_t tmem = lane_tmem_open<C::TM>(smem);
    const LaneL L = lane_view(blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, NG = (blockDim.x >> 5) / K;
    const LaneS S = lane_scratch<K, C::TM>(reinterpret_cast<float*>(blob + a.blob_bytes), L, warp, lane,
                                           lane_group_floats(L.Npad, L.own_floats, L.R, K, C::TM, C::ST), tmem);
    const int Gn = 7 + L.R, D = 6 + L.R;
    const size_t tid = ((size_t)blockIdx.x * NG + S.gid) * 32 + lane, T = (size_t)gridDim.x * NG * 32;
    const bool act = tid < (size_t)a.n;
    const size_t idx = act ? tid : (size_t)a.n - 1;
    if (S.part == 0)
        for (int d = 0; d < Gn; ++d) S.geno[d * 32] = a.genos[idx * a.gstride + d];
    group_sync<K>(S);
    LaneLS ls;
    if (C::ST) { ls.best = S.state; ls.Eg2 = ls.best + Gn * 32; ls.Ed2 = ls.Eg2 + D * 32; ls.stride = 32; }
    else { ls.best = scratch + tid; ls.Eg2 = ls.best + (size_t)Gn * T; ls.Ed2 = ls.Eg2 + (size_t)D * T; ls.stride = (int)T; }
    int iters = 0;
    float* tr = a.trace ? a.trace + idx * P.lsit : nullptr;
    const float e = SW ? lane_solis_wets<K, C::TM>(L, G, P, S, ls, act, (act && S.part == 0) ? a.E[idx] : 0.f, a.seed, (uint32_t)idx, a.gen, iters, tr, 1)
                       : lane_adadelta<K, C::TM>(L, G, P, S, ls, act, __int_as_float(0x7fc00000), iters, tr, 1);
    if (act && S.part == 0) {
        for (int d = 0; d < Gn; ++d) a.genos[idx * a.gstride + d] = ls.best[(size_t)d * ls.stride];
        a.E[idx] = e;
        if (a.iters) a.iters[idx] = iters;
    }
    lane_tmem_close<C::TM>(tmem);
}

template <class C, bool SW>
static int launch_ls_array_lane(const adock_grids* grids, const adock_ligand* ligand, const ParDev& P, LsArgs a, int var, int n, cudaStream_t stm) {
    const LaneGeom g = lane_geom(ligand);
    const int ngroups = (n + 31) / 32;
    const int NG = lane_spread_groups(lane_fit_groups(g, var, true), ngroups, C::K);
    const int grid = (ngroups + NG - 1) / NG;
    const size_t smem = lane_smem(g, var, true, NG);
    const size_t T = (size_t)grid * NG * 32;
    const int R = ligand->tp.R;
    float* scratch = nullptr;
    cudaError_t e = cudaMallocAsync(&scratch, C::ST ? 16 : T * (size_t)(7 + R + 2 * (6 + R)) * 4, stm);
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("ls scratch: ") + cudaGetErrorString(e));
    e = cudaFuncSetAttribute(ls_array_lane_kernel<C, SW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) {
        ls_array_lane_kernel<C, SW><<<grid, NG * C::K * 32, smem, stm>>>(grids->dev, P, a, scratch);
        ++g_launches;
        e = cudaGetLastError();
    }
    cudaFreeAsync(scratch, stm);
    if (e != cudaSuccess) return fail(ADOCK_ECUDA, std::string("ls_array_lane_kernel: ") + cudaGetErrorString(e));
    return ADOCK_OK;
}

// method: 0 = ADADELTA, 1 = Solis-Wets (d_energies then carries the starting energies in)
static int local_search_impl(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params, int method,
                             float* d_genotypes, int n, int gstride, float* d_energies, int* d_iters, float* d_trace,
                             unsigned long long seed, unsigned int gen, void* cuda_stream) {
    if (!grids || !ligand) return fail(ADOCK_EINVAL, "NULL handle");
    if (n < 0) return fail(ADOCK_EINVAL, "n < 0");
    if (n == 0) return ADOCK_OK;
    if (!d_genotypes || !d_energies || gstride < 7 + ligand->tp.R) return fail(ADOCK_EINVAL, "bad buffer");
    adock_params p;
    int rc = check_params(params, ligand, p);
    if (rc) return rc;
    p.ls_method = method;
    rc = device_props();
    if (rc) return rc;
    if (g_path == 2 || (g_path == 0 && n >= lane_min_chains() && lane_ok(ligand))) {
        const int var = lane_pick_var(lane_geom(ligand), (n + 31) / 32, true);
        if (var < 0) return fail(ADOCK_ELIMIT, "ligand does not fit the lane-per-individual kernel");
        ParDev P = make_pardev(p);
        P.k_wall_h = p.k_wall * grids->dev.h;
        LsArgs a{ligand->d_lane, d_genotypes, d_energies, d_iters, d_trace, ligand->lane_bytes, n, gstride, seed, gen};
        cudaStream_t stm = (cudaStream_t)cuda_stream;
        if (method == 1) { LANE_VARIANT(var, rc = launch_ls_array_lane<C, true>(grids, ligand, P, a, var, n, stm)) }
        else { LANE_VARIANT(var, rc = launch_ls_array_lane<C, false>(grids, ligand, P, a, var, n, stm)) }
        return rc;
    }
    if (g_path == 3 && method == 0) {                   // the team family's ADADELTA chain, as the docking runs it (same choice of teams per CTA)
        const size_t team = (size_t)team_scratch_floats(ligand->tp.N, ligand->tp.nfrag, ligand->tp.R);
        const size_t one = 16 + (size_t)ligand->blob_bytes + team * 4, four = 16 + (size_t)ligand->blob_bytes + 4 * team * 4;
        const int tpc = (5 * one <= (size_t)g_smem_optin || four > (size_t)g_smem_optin) ? 1 : 4;
        const size_t smem_team = tpc == 1 ? one : four;
        if (smem_team <= (size_t)g_smem_optin) {
            ParDev P = make_pardev(p);
            P.k_wall_h = p.k_wall * grids->dev.h;
            LsArgs a{ligand->d_blob, d_genotypes, d_energies, d_iters, d_trace, ligand->blob_bytes, n, gstride, seed, gen};
            if (tpc == 1) {
                CUDA_TRY(cudaFuncSetAttribute(ls_array_team_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_team));
                ls_array_team_kernel<1><<<n, kTeamW * 32, smem_team, (cudaStream_t)cuda_stream>>>(grids->dev, P, a, (int)team);
            } else {
                CUDA_TRY(cudaFuncSetAttribute(ls_array_team_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_team));
                ls_array_team_kernel<4><<<(n + 3) / 4, 4 * kTeamW * 32, smem_team, (cudaStream_t)cuda_stream>>>(grids->dev, P, a, (int)team);
            }
            ++g_launches;
            CUDA_TRY(cudaGetLastError());
            return ADOCK_OK;
        }
    }
    const int W = fit_warps(ligand->blob_bytes, ligand->scratch_floats, 4);
    if (!W) return fail(ADOCK_ELIMIT, "ligand does not fit in shared memory");
    const size_t smem = cta_smem(ligand->blob_bytes, ligand->scratch_floats, W);
    CUDA_TRY(cudaFuncSetAttribute(ls_array_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ParDev P = make_pardev(p);
    P.k_wall_h = p.k_wall * grids->dev.h;
    LsArgs a{ligand->d_blob, d_genotypes, d_energies, d_iters, d_trace, ligand->blob_bytes, n, gstride, seed, gen};
    ls_array_kernel<<<(n + W - 1) / W, W * 32, smem, (cudaStream_t)cuda_stream>>>(grids->dev, P, a);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return ADOCK_OK;
}

extern "C" int adock_local_search(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                                  float* d_genotypes, int n, int gstride, float* d_energies, int* d_iters, float* d_trace,
                                  void* cuda_stream) {
    return local_search_impl(grids, ligand, params, 0, d_genotypes, n, gstride, d_energies, d_iters, d_trace, 0ull, 0u, cuda_stream);
}

extern "C" int adock_solis_wets(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                                float* d_genotypes, int n, int gstride, float* d_energies, int* d_evals, float* d_trace,
                                unsigned long long seed, unsigned int generation, void* cuda_stream) {
    return local_search_impl(grids, ligand, params, 1, d_genotypes, n, gstride, d_energies, d_evals, d_trace, seed, generation, cuda_stream);
}

// ---- ADADELTA local search without any device allocation (callers that may not call cudaMalloc: stream capture, serving
// loops).  The chain-state columns of ls_array_lane_kernel (best genotype, E[g^2], E[dx^2]: 19 + 3R floats per chain) live
// in a file-scope device array instead of a cudaMallocAsync block.  Every GPU that loads the library holds the array until
// exit; every call shares it and finds the last call's contents there (the kernel initialises every column it reads, so
// nothing has to be cleared); calls that overlap on the GPU race on it.
static __device__ __align__(256) float g_noalloc_scratch[ADOCK_NOALLOC_SCRATCH_BYTES / 4];
static constexpr int kNoAllocMaxDevices = 64;
static float* g_noalloc_ptr[kNoAllocMaxDevices];        // device address of g_noalloc_scratch on device d (the name itself is a host-side stand-in)

// once per device, with that device current
static int noalloc_scratch_address(float** out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(ADOCK_ELIMIT, "device ordinal beyond the no-allocation path's table");
    if (!g_noalloc_ptr[dev]) {
        float* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return fail(ADOCK_ECUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e));
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return ADOCK_OK;
}

extern "C" int adock_local_search_noalloc(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                                          float* d_genotypes, int n, int gstride, float* d_energies, int* d_iters, float* d_trace,
                                          void* cuda_stream) {
    if (!grids || !ligand) return fail(ADOCK_EINVAL, "NULL handle");
    if (n < 0) return fail(ADOCK_EINVAL, "n < 0");
    if (n == 0) return ADOCK_OK;
    if (!d_genotypes || !d_energies || gstride < 7 + ligand->tp.R) return fail(ADOCK_EINVAL, "bad buffer");
    adock_params p;
    int rc = check_params(params, ligand, p);
    if (rc) return rc;
    p.ls_method = 0;
    rc = device_props();
    if (rc) return rc;
    using C = LaneCfg<1, 8, false>;                     // variant 0: positions in shared memory, chain state in global columns
    static_assert(!C::ST, "the no-allocation path is the variant whose chain state is in global scratch");
    const LaneGeom g = lane_geom(ligand);
    const int fit = lane_fit_groups(g, 0, true);
    if (fit < 1) return fail(ADOCK_ELIMIT, "ligand does not fit the lane-per-individual kernel");
    const int ngroups = (n + 31) / 32;
    const int NG = lane_spread_groups(fit, ngroups, C::K);
    const int grid = (ngroups + NG - 1) / NG;
    const size_t T = (size_t)grid * NG * 32;            // chains of the launch, padded to whole CTAs
    const int R = ligand->tp.R;
    const size_t need = T * (size_t)(7 + R + 2 * (6 + R)) * 4;
    if (need > (size_t)ADOCK_NOALLOC_SCRATCH_BYTES)
        return fail(ADOCK_ELIMIT, "adock_local_search_noalloc: " + std::to_string(n) + " chains of " + std::to_string(R) + " torsions need " +
                                      std::to_string(need) + " bytes of chain state, more than ADOCK_NOALLOC_SCRATCH_BYTES (" +
                                      std::to_string((size_t)ADOCK_NOALLOC_SCRATCH_BYTES) + "): split the batch");
    float* scratch = nullptr;
    rc = noalloc_scratch_address(&scratch);
    if (rc) return rc;
    ParDev P = make_pardev(p);
    P.k_wall_h = p.k_wall * grids->dev.h;
    LsArgs a{ligand->d_lane, d_genotypes, d_energies, d_iters, d_trace, ligand->lane_bytes, n, gstride, 0ull, 0u};
    const size_t smem = lane_smem(g, 0, true, NG);
    CUDA_TRY(cudaFuncSetAttribute(ls_array_lane_kernel<C, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ls_array_lane_kernel<C, false><<<grid, NG * C::K * 32, smem, (cudaStream_t)cuda_stream>>>(grids->dev, P, a, scratch);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    return ADOCK_OK;
}

// =================================================================== LGA docking (rows a5-a7)
struct RunState {           // 32 bytes
    long long evals;
    int gen, cur, active, ls_acc;
    int pad[2];
};
struct DockJob {
    const unsigned char* blob;
    const int* ext_of_int;
    float* pop;             // [2][nrun][P][Gn]
    float* E;               // [2][nrun][P]
    RunState* st;           // [nrun]
    int* picks;             // [nrun][P]
    int* fy;                // [nrun][P] Fisher-Yates scratch
    float* out_geno;        // [nrun][gstride]
    float* out_E;           // [nrun]
    float* out_xyz;         // [nrun][cstride][3] or NULL
    long long* out_evals;   // [nrun]
    int* out_gens;          // [nrun]
    unsigned long long seed;
    int blob_bytes, Gn, N, R;
    const unsigned char* lane;  // lane-per-individual image (lane_image.hpp)
    int lane_bytes, pad0;
    float* hist;            // [nrun][as_window] ring of each run's best energy per generation (R12 autostop) or NULL
    int* act;               // act[0] = number of active runs, act[1 + k] = k-th active run (ascending): the lane kernels
                            // deal their lanes out over the active runs only (runs end at different generations)
};
struct DockDims {
    int nrun, P, n_ls, upj;         // upj = CTAs per job for this launch
    long long max_evals;
    int max_gens, gstride, cstride;
    int autostop, as_window;        // R12
    float as_tol;
};

#define DOCK_PROLOGUE(WARPS_EXPR)                                                                                         \
    extern __shared__ __align__(128) unsigned char smem[];                                                               \
    const DockJob job = jobs[blockIdx.x / dm.upj];                                                                       \
    unsigned char* blob = smem + 16;                                                                                     \
    stage_ligand(blob, job.blob, job.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);                                  \
    const LigS L = lig_view(blob);                                                                                       \
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;                                     \
    const WarpS S = warp_view(reinterpret_cast<float*>(blob + job.blob_bytes) + (size_t)warp * warp_scratch_floats(L.N, L.nfrag, L.R), L); \
    const int ind = (blockIdx.x % dm.upj) * W + warp;                                                                    \
    const int Gn = job.Gn;                                                                                               \
    (void)Gn; (void)S; (void)lane;

// generation 0: random population + its energies; run bookkeeping
__global__ void __launch_bounds__(256) dock_init_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs, DockDims dm) {
    DOCK_PROLOGUE()
    if (ind >= dm.nrun * dm.P) return;
    const int run = ind / dm.P, slot = ind % dm.P;
    ga_init_individual(G, L.R, job.seed, (uint32_t)ind, S.geno, lane);
    __syncwarp();
    float* dst = job.pop + (size_t)ind * Gn;
    for (int d = lane; d < Gn; d += 32) dst[d] = S.geno[d];
    float ei, ea;
    const float e = eval_pose<false>(L, G, P, S, lane, ei, ea);
    if (lane == 0) {
        job.E[ind] = e;
        if (slot == 0) {
            RunState s;
            s.evals = dm.P; s.gen = 0; s.cur = 0; s.ls_acc = 0; s.pad[0] = s.pad[1] = 0;
            s.active = (s.evals < dm.max_evals && dm.max_gens > 0) ? 1 : 0;
            job.st[run] = s;
        }
    }
}

// one GA generation: elitism, tournament selection, two-point crossover, mutation, scoring of the offspring;
// the slot-0 warp also draws this generation's local-search subset
template <bool SCORE>
__global__ void __launch_bounds__(256) dock_ga_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs, DockDims dm,
                                                      int* __restrict__ decisions) {
    DOCK_PROLOGUE()
    if (ind >= dm.nrun * dm.P) return;
    const int run = ind / dm.P, slot = ind % dm.P;
    const RunState st = job.st[run];
    if (!st.active) return;
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const float* spop = job.pop + ((size_t)st.cur * popsz + (size_t)run * dm.P) * Gn;
    const float* sE = job.E + (size_t)st.cur * popsz + (size_t)run * dm.P;
    float* dpop = job.pop + ((size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P) * Gn;
    float* dE = job.E + (size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P;
    const uint32_t gen = (uint32_t)st.gen + 1u;
    int* dec = decisions ? decisions + ((size_t)(blockIdx.x / dm.upj) * popsz + ind) * 10 : nullptr;
    if (slot == 0) {
        float be = __int_as_float(0x7f800000);
        int bi = 0x7fffffff;
        for (int s = lane; s < dm.P; s += 32) {
            const float e = sE[s];
            if (e < be) { be = e; bi = s; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float oe = __shfl_xor_sync(kFull, be, o);
            const int oi = __shfl_xor_sync(kFull, bi, o);
            if (oe < be || (oe == be && oi < bi)) { be = oe; bi = oi; }
        }
        if (bi == 0x7fffffff) bi = 0;                    // every energy non-finite: keep slot 0
        for (int d = lane; d < Gn; d += 32) dpop[d] = spop[(size_t)bi * Gn + d];
        if (lane == 0) {
            dE[0] = sE[bi];
            if (dec) { for (int k = 0; k < 10; ++k) dec[k] = 0; dec[2] = bi; }
        }
        // local-search subset: slot 0 + first n_ls-1 entries of a partial Fisher-Yates shuffle of 1..P-1
        int* picks = job.picks + (size_t)run * dm.P;
        if (dm.n_ls >= dm.P) {
            for (int s = lane; s < dm.P; s += 32) picks[s] = s;
        } else if (dm.n_ls > 0) {
            int* fy = job.fy + (size_t)run * dm.P;
            for (int s = lane; s < dm.P - 1; s += 32) fy[s] = s + 1;
            __syncwarp();
            if (lane == 0) {
                picks[0] = 0;
                uint4 r = make_uint4(0, 0, 0, 0);
                for (int m = 0; m < dm.n_ls - 1; ++m) {
                    if ((m & 3) == 0) r = draw4(job.seed, (uint32_t)(m >> 2), kLsPick, (uint32_t)(run * dm.P), gen);
                    const int j = m + below(pick_word(r, m & 3), dm.P - 1 - m);
                    const int t = fy[m]; fy[m] = fy[j]; fy[j] = t;
                    picks[1 + m] = fy[m];
                }
            }
        }
        return;
    }
    ga_make_child(P, dm.P, L.R, job.seed, (uint32_t)ind, gen, spop, sE, S.geno, dec, lane);
    for (int d = lane; d < Gn; d += 32) dpop[(size_t)slot * Gn + d] = S.geno[d];
    if (SCORE) {
        float ei, ea;
        const float e = eval_pose<false>(L, G, P, S, lane, ei, ea);
        if (lane == 0) dE[slot] = e;
    }
}

// The same generation step with a THREAD per individual of the new population (no shared memory, no ligand image): the
// warp-per-offspring kernel above spends a warp on work that is a dozen Philox draws (1.5 ms per generation for 592 ligands);
// here the thread of slot 0 copies the elite and draws the local-search subset, every other thread makes its child
// (ga_make_child_thread: bit-identical to ga_make_child).  Used with the lane-per-individual offspring scoring.
__global__ void __launch_bounds__(128) dock_ga_lane_kernel(ParDev P, const DockJob* __restrict__ jobs, DockDims dm, int* __restrict__ decisions) {
    const DockJob& job = jobs[blockIdx.x / dm.upj];
    const int ind = (blockIdx.x % dm.upj) * blockDim.x + threadIdx.x;
    if (ind >= dm.nrun * dm.P) return;
    const int run = ind / dm.P, slot = ind % dm.P, Gn = job.Gn;
    const RunState st = job.st[run];
    if (!st.active) return;
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const float* spop = job.pop + ((size_t)st.cur * popsz + (size_t)run * dm.P) * Gn;
    const float* sE = job.E + (size_t)st.cur * popsz + (size_t)run * dm.P;
    float* dpop = job.pop + ((size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P) * Gn;
    float* dE = job.E + (size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P;
    const uint32_t gen = (uint32_t)st.gen + 1u;
    int* dec = decisions ? decisions + ((size_t)(blockIdx.x / dm.upj) * popsz + ind) * 10 : nullptr;
    if (slot == 0) {
        float be = __int_as_float(0x7f800000);
        int bi = 0x7fffffff;
        for (int s = 0; s < dm.P; ++s) {                // ties: the lowest slot (strict <, ascending)
            const float e = sE[s];
            if (e < be) { be = e; bi = s; }
        }
        if (bi == 0x7fffffff) bi = 0;                    // every energy non-finite: keep slot 0
        for (int d = 0; d < Gn; ++d) dpop[d] = spop[(size_t)bi * Gn + d];
        dE[0] = sE[bi];
        if (dec) { for (int k = 0; k < 10; ++k) dec[k] = 0; dec[2] = bi; }
        int* picks = job.picks + (size_t)run * dm.P;
        if (dm.n_ls >= dm.P) {
            for (int s = 0; s < dm.P; ++s) picks[s] = s;
        } else if (dm.n_ls > 0) {
            int* fy = job.fy + (size_t)run * dm.P;
            for (int s = 0; s < dm.P - 1; ++s) fy[s] = s + 1;
            picks[0] = 0;
            uint4 r = make_uint4(0, 0, 0, 0);
            for (int m = 0; m < dm.n_ls - 1; ++m) {
                if ((m & 3) == 0) r = draw4(job.seed, (uint32_t)(m >> 2), kLsPick, (uint32_t)(run * dm.P), gen);
                const int j = m + below(pick_word(r, m & 3), dm.P - 1 - m);
                const int t = fy[m]; fy[m] = fy[j]; fy[j] = t;
                picks[1 + m] = fy[m];
            }
        }
        return;
    }
    ga_make_child_thread(P, dm.P, job.R, job.seed, (uint32_t)ind, gen, spop, sE, dpop + (size_t)slot * Gn, dec);
}

// ADADELTA on the selected individuals of the new population (Lamarckian write-back)
__global__ void __launch_bounds__(128) dock_ls_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs, DockDims dm) {
    DOCK_PROLOGUE()
    if (ind >= dm.nrun * dm.n_ls) return;
    const int run = ind / dm.n_ls, l = ind % dm.n_ls;
    const RunState st = job.st[run];
    if (!st.active) return;
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const int slot = job.picks[(size_t)run * dm.P + l];
    float* g = job.pop + ((size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P + slot) * Gn;
    float* e = job.E + (size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P + slot;
    for (int d = lane; d < Gn; d += 32) S.geno[d] = g[d];
    __syncwarp();
    int iters = 0;
    const float be = P.ls_method == 1
                         ? solis_wets_search(L, G, P, S, lane, *e, job.seed, (uint32_t)(run * dm.P + slot), (uint32_t)st.gen + 1u, iters)
                         : adadelta_search(L, G, P, S, lane, *e, iters);
    for (int d = lane; d < Gn; d += 32) g[d] = S.best[d];
    if (lane == 0) {
        *e = be;
        atomicAdd(&job.st[run].ls_acc, iters);
    }
}

// ADADELTA with one TEAM (kTeamW warps) per chain: launches with too few chains to give every scheduler a warp.
// TPC teams share a CTA and its ligand image.  TPC = 1: 5 CTAs per SM (<= 102 registers): 4 ligands x 180 chains are one
// wave; at 4 CTAs per SM they were two (1.85 s -> 3.08 s).  TPC = 4 (one CTA per SM, <= 128 registers): ligands whose image
// fills most of the shared memory (128 atoms: 117 KB of pair records), where one team per CTA left three of the four
// schedulers of an SM without a warp.
#ifndef TEAM_NF1
#define TEAM_NF1 2
#endif
#ifndef TEAM_NF4
#define TEAM_NF4 4
#endif
template <int TPC>
__global__ void __launch_bounds__(TPC * kTeamW * 32, TPC == 1 ? 5 : 1) dock_ls_team_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs,
                                                                                          DockDims dm, int team_floats) {
    extern __shared__ __align__(128) unsigned char smem[];
    const DockJob job = jobs[blockIdx.x / dm.upj];
    unsigned char* blob = smem + 16;
    stage_ligand(blob, job.blob, job.blob_bytes, reinterpret_cast<uint64_t*>(smem), 0);
    const LigS L = lig_view(blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int team = warp / kTeamW;
    TeamS T = team_view(reinterpret_cast<float*>(blob + job.blob_bytes) + (size_t)team * team_floats, L, warp % kTeamW);
    T.bar = 1 + team;
    const int ind = (blockIdx.x % dm.upj) * TPC + team, Gn = job.Gn;
    if (ind >= dm.nrun * dm.n_ls) return;               // whole teams leave: the barriers below are per team
    const int run = ind / dm.n_ls, l = ind % dm.n_ls;
    const RunState st = job.st[run];
    if (!st.active) return;
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const int slot = job.picks[(size_t)run * dm.P + l];
    float* g = job.pop + ((size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P + slot) * Gn;
    float* e = job.E + (size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P + slot;
    if (T.wi == 0) for (int d = lane; d < Gn; d += 32) T.S.geno[d] = g[d];
    team_sync(T);
    int iters = 0;
    const float be = adadelta_search_team<TPC == 1 ? TEAM_NF1 : TEAM_NF4, TPC == 4>(L, G, P, T, lane, *e, iters);
    if (T.wi == 0) {
        for (int d = lane; d < Gn; d += 32) g[d] = T.S.best[d];
        if (lane == 0) {
            *e = be;
            atomicAdd(&job.st[run].ls_acc, iters);
        }
    }
}

// ---- lane-per-individual kernels of the docking loop.  The groups (32 chains / individuals each) of all jobs of a
// launch form one flat sequence, jg groups per job; CTA b takes groups [b*ng, (b+1)*ng), which may belong to several
// consecutive jobs: it stages the lane image of each of them (slot s = job j0+s) in one bulk-copy transaction.
struct LaneDockArgs {
    float* scratch;         // ADADELTA state columns (LS kernel)
    int Gmax;               // largest 7+R of the launch
    int ng, total_groups, jg;
    int slot_bytes, nimg;   // image slots per CTA (the most any CTA needs), slot size (multiple of 128)
    int group_floats;       // floats per lane between groups (largest ligand)
    // queue mode of the local-search kernel (dock_ls_lane_queue_kernel): a CTA holds `tpc` teams of `jg` groups; team T of the
    // launch docks the jobs q_job[q_off[T] .. q_off[T+1]) one after the other
    int tpc;
    const int* q_off;
    const int* q_job;
};
constexpr int kLaneQueueHeader = 128;     // bulk-copy barrier of team t at byte 16 + 8 t (t < 7); tensor-memory address at byte 8
constexpr int kLaneQueueMaxTeams = 7;
struct LaneCtaGroup { int jidx, gi; const unsigned char* blob; float* scratch; bool valid; };
template <int K>
__device__ __forceinline__ LaneCtaGroup lane_cta_group(unsigned char* smem, const DockJob* __restrict__ jobs, const LaneDockArgs& a) {
    const int first = blockIdx.x * a.ng, last = min(first + a.ng, a.total_groups) - 1;
    const int j0 = first / a.jg, nimg = last / a.jg - j0 + 1;
    stage_images(smem + 16, a.slot_bytes, nimg,
                 [&](int s, const unsigned char*& p, int& b) { p = jobs[j0 + s].lane; b = jobs[j0 + s].lane_bytes; },
                 reinterpret_cast<uint64_t*>(smem));
    LaneCtaGroup c;
    const int g = first + (int)(threadIdx.x >> 5) / K;
    c.valid = g <= last;
    c.jidx = c.valid ? g / a.jg : j0;
    c.gi = c.valid ? g % a.jg : 0;
    c.blob = smem + 16 + (size_t)(c.jidx - j0) * a.slot_bytes;
    c.scratch = reinterpret_cast<float*>(smem + 16 + (size_t)a.nimg * a.slot_bytes);
    return c;
}

// ADADELTA on the selected individuals (Lamarckian write-back): lane c of a job's groups runs chain c = run*n_ls + l;
// ADADELTA state in global scratch columns [row][all group lanes of the launch] (rows: Gmax best, 2 x Dmax)
template <class C, bool SW>
__device__ __forceinline__ void dock_ls_lane_group(const GridDev& G, const ParDev& P, const DockJob* __restrict__ jobs, const DockDims& dm,
                                                   const LaneDockArgs& a, const LaneCtaGroup& cg, uint32_t tmem) {
    constexpr int K = C::K;
    const DockJob job = jobs[cg.jidx];
    const LaneL L = lane_view(cg.blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const LaneS S = lane_scratch<K, C::TM>(cg.scratch, L, warp, lane, a.group_floats, tmem);
    const int Gn = job.Gn;
    const int c = cg.gi * 32 + lane;
    bool act = c < job.act[0] * dm.n_ls;
    const int cc = act ? c : 0;
    const int run = job.act[1 + cc / dm.n_ls], l = cc % dm.n_ls;
    const RunState st = job.st[run];
    act = act && st.active;
    if (!__any_sync(kFull, act)) return;                // the same for every warp of the group
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const int slot = job.picks[(size_t)run * dm.P + l];
    float* g = job.pop + ((size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P + slot) * Gn;
    float* e = job.E + (size_t)(st.cur ^ 1) * popsz + (size_t)run * dm.P + slot;
    if (S.part == 0)
        for (int d = 0; d < Gn; ++d) S.geno[d * 32] = g[d];
    group_sync<K>(S);
    const size_t tid = ((size_t)blockIdx.x * a.ng + S.gid) * 32 + lane, T = (size_t)gridDim.x * a.ng * 32;
    const int Dmax = a.Gmax - 1;
    LaneLS ls;
    if (C::ST) { ls.best = S.state; ls.Eg2 = ls.best + Gn * 32; ls.Ed2 = ls.Eg2 + (Gn - 1) * 32; ls.stride = 32; }
    else { ls.best = a.scratch + tid; ls.Eg2 = ls.best + (size_t)a.Gmax * T; ls.Ed2 = ls.Eg2 + (size_t)Dmax * T; ls.stride = (int)T; }
    int iters = 0;
    const float e0 = (act && S.part == 0) ? *e : 0.f;
    const float be = SW ? lane_solis_wets<K, C::TM>(L, G, P, S, ls, act, e0, job.seed, (uint32_t)(run * dm.P + slot), (uint32_t)st.gen + 1u, iters, nullptr, 0)
                        : lane_adadelta<K, C::TM>(L, G, P, S, ls, act, e0, iters, nullptr, 0);
    if (act && S.part == 0) {
        for (int d = 0; d < Gn; ++d) g[d] = ls.best[(size_t)d * ls.stride];
        *e = be;
        atomicAdd(&job.st[run].ls_acc, iters);
    }
}
template <class C, bool SW>
__global__ void __launch_bounds__(C::kMaxWarps * 32, 1) dock_ls_lane_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs, DockDims dm,
                                                                            LaneDockArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const LaneCtaGroup cg = lane_cta_group<C::K>(smem, jobs, a);
    const uint32_t tmem = lane_tmem_open<C::TM>(smem);
    if (cg.valid) dock_ls_lane_group<C, SW>(G, P, jobs, dm, a, cg, tmem);     // whole groups skip: the named barriers are per group
    lane_tmem_close<C::TM>(tmem);
}

// The same with a work queue per TEAM (the jg groups of one ligand: one image slot).  The flat partition above gives every
// group slot exactly one group, so a launch lasts as long as its heaviest ligand and the slots of the light ones idle; here
// the host deals the ligands of the launch (two or three per team) to the teams by estimated cost, longest first, and a
// team stages the next ligand's image itself (bulk copy into its slot, its own mbarrier and named barrier) when it is done
// with the previous one: the teams of a CTA never wait for each other.
template <class C, bool SW>
__global__ void __launch_bounds__(C::kMaxWarps * 32, 1) dock_ls_lane_queue_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs,
                                                                                  DockDims dm, LaneDockArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tw = a.jg * C::K;                         // warps per team
    const int team = warp / tw, wt = warp % tw;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 16) + team;
    const bool leader = wt == 0 && lane == 0;
    if (leader) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t tmem = lane_tmem_open<C::TM>(smem);
    unsigned char* slot = smem + kLaneQueueHeader + (size_t)team * a.slot_bytes;
    float* scratch = reinterpret_cast<float*>(smem + kLaneQueueHeader + (size_t)a.tpc * a.slot_bytes);
    const int T = blockIdx.x * a.tpc + team;
    uint32_t phase = 0;
    for (int q = a.q_off[T]; q < a.q_off[T + 1]; ++q) {
        const int jidx = a.q_job[q];
        if (leader) {
            const int bytes = jobs[jidx].lane_bytes;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(slot)),
                         "l"(jobs[jidx].lane), "r"(bytes), "r"(smem_u32(bar))
                         : "memory");
        }
        uint32_t done = 0;
        while (!done) {
            asm volatile(
                "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                : "=r"(done)
                : "r"(smem_u32(bar)), "r"(phase)
                : "memory");
        }
        phase ^= 1u;
        const LaneCtaGroup cg{jidx, wt / C::K, slot, scratch, true};
        dock_ls_lane_group<C, SW>(G, P, jobs, dm, a, cg, tmem);
        asm volatile("bar.sync %0, %1;" ::"r"(9 + team), "r"(tw * 32) : "memory");       // the team is done with this image
    }
    lane_tmem_close<C::TM>(tmem);
}

// energies of the offspring written by dock_ga_kernel<false> (slot 0, the elite, carries its energy): lane c of a
// job's groups scores individual c = run*P + slot of the new population
template <class C>
__device__ __forceinline__ void dock_score_lane_group(const GridDev& G, const ParDev& P, const DockJob* __restrict__ jobs, const DockDims& dm,
                                                      const LaneDockArgs& a, const LaneCtaGroup& cg, uint32_t tmem) {
    constexpr int K = C::K;
    const DockJob job = jobs[cg.jidx];
    const LaneL L = lane_view(cg.blob);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const LaneS S = lane_scratch<K, C::TM>(cg.scratch, L, warp, lane, a.group_floats, tmem);
    const int Gn = job.Gn;
    const int c = cg.gi * 32 + lane, n = job.act[0] * dm.P;
    bool act = c < n;
    const int ca = act ? c : 0;
    const int run = job.act[1 + ca / dm.P], slot = ca % dm.P;
    const int cc = run * dm.P + slot;
    const RunState st = job.st[run];
    act = act && st.active && slot != 0;
    if (!__any_sync(kFull, act)) return;
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const float* g = job.pop + ((size_t)(st.cur ^ 1) * popsz + cc) * Gn;
    if (S.part == 0)
        for (int d = 0; d < Gn; ++d) S.geno[d * 32] = g[d];
    group_sync<K>(S);
    float ei, ea;
    bool gf;
    const float e = lane_eval<false, K, 1, C::TM>(L, G, P, S, nullptr, 1, false, ei, ea, gf);
    if (act && S.part == 0) job.E[(size_t)(st.cur ^ 1) * popsz + cc] = e;
}
template <class C>
__global__ void __launch_bounds__(C::kMaxWarps * 32, 1) dock_score_lane_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs, DockDims dm,
                                                                               LaneDockArgs a) {
    extern __shared__ __align__(128) unsigned char smem[];
    const LaneCtaGroup cg = lane_cta_group<C::K>(smem, jobs, a);
    const uint32_t tmem = lane_tmem_open<C::TM>(smem);
    if (cg.valid) dock_score_lane_group<C>(G, P, jobs, dm, a, cg, tmem);
    lane_tmem_close<C::TM>(tmem);
}

// end of generation: eval accounting, buffer flip, termination test
// one CTA per job, threads over its runs; thread 0 then rebuilds the job's list of active runs
__device__ __forceinline__ void dock_commit_run(const DockJob& job, int run, const DockDims& dm, int* __restrict__ any_active);
__global__ void __launch_bounds__(128) dock_commit_kernel(const DockJob* __restrict__ jobs, int njobs, DockDims dm, int* __restrict__ any_active) {
    const DockJob& job = jobs[blockIdx.x];
    for (int run = threadIdx.x; run < dm.nrun; run += blockDim.x) dock_commit_run(job, run, dm, any_active);
    __syncthreads();
    if (threadIdx.x == 0) {
        int n = 0;
        for (int run = 0; run < dm.nrun; ++run)
            if (job.st[run].active) job.act[1 + n++] = run;
        job.act[0] = n;
    }
}
__device__ __forceinline__ void dock_commit_run(const DockJob& job, int run, const DockDims& dm, int* __restrict__ any_active) {
    RunState* s = job.st + run;
    if (!s->active) return;
    s->evals += (long long)(dm.P - 1) + s->ls_acc;
    s->ls_acc = 0;
    s->gen += 1;
    s->cur ^= 1;
    bool stop = false;
    if (dm.autostop) {              // R12: std-dev of the run's best energy over the last as_window generations < as_tol
        const int W = dm.as_window;
        const float* E = job.E + ((size_t)s->cur * dm.nrun + run) * dm.P;
        float best = E[0];
        for (int k = 1; k < dm.P; ++k) best = fminf(best, E[k]);
        float* h = job.hist + (size_t)run * W;
        h[(s->gen - 1) % W] = best;
        if (s->gen >= W) {
            float m = 0.f, v = 0.f;
            for (int k = 0; k < W; ++k) m += h[k];
            m /= (float)W;
            for (int k = 0; k < W; ++k) { const float d = h[k] - m; v += d * d; }
            stop = sqrtf(v / (float)W) < dm.as_tol;
        }
    }
    s->active = (!stop && s->evals < dm.max_evals && s->gen < dm.max_gens) ? 1 : 0;
    if (s->active) atomicOr(any_active, 1);
}

// per run: best individual of the final population, its pose in the caller's atom order
__global__ void __launch_bounds__(128) dock_final_kernel(GridDev G, ParDev P, const DockJob* __restrict__ jobs, DockDims dm) {
    DOCK_PROLOGUE()
    if (ind >= dm.nrun) return;
    const int run = ind;
    const RunState st = job.st[run];
    const size_t popsz = (size_t)dm.nrun * dm.P;
    const float* pop = job.pop + ((size_t)st.cur * popsz + (size_t)run * dm.P) * Gn;
    const float* E = job.E + (size_t)st.cur * popsz + (size_t)run * dm.P;
    float be = __int_as_float(0x7f800000);
    int bi = 0x7fffffff;
    for (int s = lane; s < dm.P; s += 32) {
        const float e = E[s];
        if (e < be) { be = e; bi = s; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float oe = __shfl_xor_sync(kFull, be, o);
        const int oi = __shfl_xor_sync(kFull, bi, o);
        if (oe < be || (oe == be && oi < bi)) { be = oe; bi = oi; }
    }
    if (bi == 0x7fffffff) bi = 0;
    for (int d = lane; d < Gn; d += 32) {
        const float v = pop[(size_t)bi * Gn + d];
        S.geno[d] = v;
        job.out_geno[(size_t)run * dm.gstride + d] = v;
    }
    __syncwarp();
    float ei, ea;
    eval_pose<false>(L, G, P, S, lane, ei, ea);
    if (job.out_xyz)
        for (int i = lane; i < L.npos; i += 32) {
            const int e = job.ext_of_int[i];
            if (e < 0) continue;
            const float* b = S.blk + atom_slot_dev(i);
            float* o = job.out_xyz + ((size_t)run * dm.cstride + e) * 3;
            o[0] = b[kX]; o[1] = b[kY]; o[2] = b[kZ];
        }
    if (lane == 0) {
        job.out_E[run] = E[bi];
        job.out_evals[run] = st.evals;
        job.out_gens[run] = st.gen;
    }
}

namespace {
struct DevBuf {             // frees on scope exit
    std::vector<void*> ptrs;
    ~DevBuf() { for (void* p : ptrs) cudaFree(p); }
    template <class T> cudaError_t alloc(T** p, size_t n) {
        cudaError_t e = cudaMalloc((void**)p, n ? n : 1);
        if (e == cudaSuccess) ptrs.push_back(*p);
        return e;
    }
};
int n_ls_of(const adock_params& p, int P) {
    int n = (int)std::ceil((double)p.lsrat * P - 1e-9);
    return std::max(0, std::min(P, n));
}
}  // namespace

static int dock_impl(const adock_grids* grids, const adock_ligand* const* ligs, int nlig, const adock_params* params, int nrun,
                     int Pn, long long max_evals, const unsigned long long* seeds, int gstride, float* best_genotypes,
                     float* best_energies, int cstride, float* best_coords, long long* evals_used, int* gens_used, cudaStream_t stm) {
    if (!grids || !ligs || !seeds || !best_genotypes || !best_energies) return fail(ADOCK_EINVAL, "NULL argument");
    if (nlig < 1 || nrun < 1 || Pn < 2 || max_evals < 0) return fail(ADOCK_EINVAL, "bad docking dimensions");
    if ((long long)nrun * Pn > (1ll << 30)) return fail(ADOCK_ELIMIT, "nrun*pop_size too large");
    int rc = device_props();
    if (rc) return rc;
    adock_params p;
    int maxblob = 0, maxscr = 0, maxteam = 0;
    for (int l = 0; l < nlig; ++l) {
        if (!ligs[l]) return fail(ADOCK_EINVAL, "NULL ligand");
        rc = check_params(params, ligs[l], p);
        if (rc) return rc;
        if (gstride < 7 + ligs[l]->tp.R || (best_coords && cstride < ligs[l]->tp.N)) return fail(ADOCK_EINVAL, "output stride too small");
        maxblob = std::max(maxblob, ligs[l]->blob_bytes);
        maxscr = std::max(maxscr, ligs[l]->scratch_floats);
        maxteam = std::max(maxteam, team_scratch_floats(ligs[l]->tp.N, ligs[l]->tp.nfrag, ligs[l]->tp.R));
    }
    const int Wga = fit_warps(maxblob, maxscr, 8), Wls = fit_warps(maxblob, maxscr, 4);
    if (!Wga || !Wls) return fail(ADOCK_ELIMIT, "ligand does not fit in shared memory");
    // local search: lane-per-individual when there are enough chains to fill the SMs with whole warps
    const int n_ls0 = n_ls_of(p, Pn);
    const long long chains = (long long)nlig * nrun * n_ls0;
    LaneGeom lg{0, 0, 0, 0};
    int Gmax = 7;
    bool lanes_fit = true;
    for (int l = 0; l < nlig; ++l) {
        lg = lane_geom_max(lg, lane_geom(ligs[l]));
        Gmax = std::max(Gmax, 7 + ligs[l]->tp.R);
        lanes_fit = lanes_fit && lane_ok(ligs[l]);
    }
    const int jg = (nrun * n_ls0 + 31) / 32;                        // groups of 32 chains per job
    const LanePlan pl = lane_plan(lg, (long long)nlig * jg, jg, true);
    // Solis-Wets chains end after very different numbers of evaluations (28 to lsit iterations), which leaves most lanes
    // of a lane-per-chain warp idle; one warp per chain is 2x faster there (profiles/r01d_next_rows.md)
    const bool many = g_path == 0 && lanes_fit && chains >= lane_min_chains();
    const bool ls_lane = pl.var >= 0 && (g_path == 2 || (many && p.ls_method == 0));
    if (g_path == 2 && pl.var < 0) return fail(ADOCK_ELIMIT, "ligand does not fit the lane-per-individual kernel");
    // a team (CTA of kTeamW warps) per chain when one warp per chain would leave most schedulers without a warp
    // teams per CTA: one where five CTAs fit an SM anyway (small images), four where the image lets only one CTA in
    const int team_tpc = (5 * (16 + (size_t)maxblob + (size_t)maxteam * 4) <= (size_t)g_smem_optin || 16 + (size_t)maxblob + 4 * (size_t)maxteam * 4 > (size_t)g_smem_optin) ? 1 : 4;
    const size_t smem_team = 16 + (size_t)maxblob + (size_t)team_tpc * maxteam * 4;
    const bool ls_team = !ls_lane && p.ls_method == 0 && smem_team <= (size_t)g_smem_optin &&
                         (g_path == 3 || (g_path == 0 && chains <= (long long)g_sm_count * 24));  // measured cross-over against warp per chain: 20 ligands x 180 chains
    g_last_dock_path = ls_lane ? 2 : ls_team ? 3 : 1;
    // offspring scoring: lane-per-individual under the same condition (populations are 1/lsrat times larger)
    const int jgs = (int)(((long long)nrun * Pn + 31) / 32);
    const LanePlan ps = lane_plan(lg, (long long)nlig * jgs, jgs, false);
    const bool ga_lane = ps.var >= 0 && (g_path == 2 || many);
    ParDev P = make_pardev(p);
    P.k_wall_h = p.k_wall * grids->dev.h;
    DockDims dm{};
    dm.nrun = nrun; dm.P = Pn; dm.n_ls = n_ls_of(p, Pn); dm.max_evals = max_evals; dm.max_gens = p.max_gens;
    dm.gstride = gstride; dm.cstride = cstride;
    dm.autostop = p.autostop; dm.as_window = p.as_window; dm.as_tol = p.as_tol;

    DevBuf buf;
    std::vector<DockJob> jobs(nlig);
    const size_t popsz = (size_t)nrun * Pn;
    float *d_out_geno = nullptr, *d_out_E = nullptr, *d_out_xyz = nullptr;
    long long* d_out_evals = nullptr;
    int *d_out_gens = nullptr, *d_flag = nullptr;
    DockJob* d_jobs = nullptr;
    // ONE device allocation per call for the outputs, the job table and every per-job buffer (device buffers are
    // preallocated, not allocated per ligand): sizes first, then the slab is carved at 256-byte boundaries
    auto up256 = [](size_t x) { return (x + 255) & ~(size_t)255; };
    size_t slab_bytes = 0;
    auto reserve = [&](size_t bytes) { const size_t o = slab_bytes; slab_bytes += up256(bytes ? bytes : 1); return o; };
    const size_t o_geno = reserve((size_t)nlig * nrun * gstride * 4), o_E = reserve((size_t)nlig * nrun * 4),
                 o_xyz = best_coords ? reserve((size_t)nlig * nrun * cstride * 12) : 0, o_evals = reserve((size_t)nlig * nrun * 8),
                 o_gens = reserve((size_t)nlig * nrun * 4), o_flag = reserve(4), o_jobs = reserve((size_t)nlig * sizeof(DockJob));
    struct JobOff { size_t pop, E, st, picks, fy, act, hist; };
    std::vector<JobOff> joff(nlig);
    for (int l = 0; l < nlig; ++l) {
        const size_t Gn = 7 + (size_t)ligs[l]->tp.R;
        joff[l] = JobOff{reserve(2 * popsz * Gn * 4), reserve(2 * popsz * 4), reserve((size_t)nrun * sizeof(RunState)), reserve(popsz * 4),
                         reserve(popsz * 4), reserve((size_t)(nrun + 1) * 4), p.autostop ? reserve((size_t)nrun * p.as_window * 4) : 0};
    }
    unsigned char* slab = nullptr;
    cudaError_t e = buf.alloc(&slab, slab_bytes);
    if (e == cudaSuccess) {
        d_out_geno = reinterpret_cast<float*>(slab + o_geno); d_out_E = reinterpret_cast<float*>(slab + o_E);
        d_out_xyz = best_coords ? reinterpret_cast<float*>(slab + o_xyz) : nullptr;
        d_out_evals = reinterpret_cast<long long*>(slab + o_evals); d_out_gens = reinterpret_cast<int*>(slab + o_gens);
        d_flag = reinterpret_cast<int*>(slab + o_flag); d_jobs = reinterpret_cast<DockJob*>(slab + o_jobs);
    }
    std::vector<int> act0(nrun + 1);                    // every run starts active
    act0[0] = nrun;
    for (int r = 0; r < nrun; ++r) act0[1 + r] = r;
    // Position of each ligand in the flat group sequence of the lane kernels: consecutive groups share a CTA, and a
    // launch lasts as long as its most loaded CTA, so heavy and light ligands alternate (sorted by estimated cost,
    // then dealt heaviest, lightest, second heaviest, ...: max/mean CTA load of the 197-ligand bench batch 1.085 -> 1.03).
    // A ligand's docking does not depend on its position (every job carries its own buffers, seed and outputs).
    std::vector<int> jorder(nlig);
    std::iota(jorder.begin(), jorder.end(), 0);
    std::vector<double> cost(nlig);
    for (int l = 0; l < nlig; ++l) {
        const LaneHeader* h = reinterpret_cast<const LaneHeader*>(ligs[l]->lane.blob.data());
        cost[l] = 56.0 * h->nrows + 160.0 * h->N + 40.0 * h->ntiles + 1500.0;
    }
    if (nlig > 2) {
        std::vector<int> by(nlig);
        std::iota(by.begin(), by.end(), 0);
        std::stable_sort(by.begin(), by.end(), [&](int a, int b) { return cost[a] > cost[b]; });
        // more CTAs than SMs: heaviest first, similar ligands share a CTA (its warps finish together) and the hardware hands
        // the next CTA to the SM that frees first -- longest-processing-time-first for free (592 bench ligands: 5.91e8 ->
        // 6.02e8 evals/s in the ADADELTA kernel); one wave: alternate, so that every CTA carries the same load
        const long long lane_ctas = pl.var >= 0 ? ((long long)nlig * jg + pl.ng - 1) / pl.ng : 0;
        if (lane_ctas > g_sm_count) jorder = by;
        else
            for (int k = 0, lo = 0, hi = nlig - 1; k < nlig; ++k) jorder[k] = (k & 1) ? by[hi--] : by[lo++];
    }
    for (int k = 0; k < nlig && e == cudaSuccess; ++k) {
        const int l = jorder[k];
        DockJob& j = jobs[k];
        const adock_ligand* lg = ligs[l];
        j.blob = lg->d_blob; j.ext_of_int = lg->d_ext_of_int; j.blob_bytes = lg->blob_bytes;
        j.Gn = 7 + lg->tp.R; j.N = lg->tp.N; j.R = lg->tp.R; j.seed = seeds[l];
        j.lane = lg->d_lane; j.lane_bytes = lg->lane_bytes; j.pad0 = 0;
        const JobOff& jo = joff[l];
        j.pop = reinterpret_cast<float*>(slab + jo.pop); j.E = reinterpret_cast<float*>(slab + jo.E);
        j.st = reinterpret_cast<RunState*>(slab + jo.st); j.picks = reinterpret_cast<int*>(slab + jo.picks);
        j.fy = reinterpret_cast<int*>(slab + jo.fy); j.act = reinterpret_cast<int*>(slab + jo.act);
        j.hist = p.autostop ? reinterpret_cast<float*>(slab + jo.hist) : nullptr;
        e = cudaMemcpyAsync(j.act, act0.data(), (size_t)(nrun + 1) * 4, cudaMemcpyHostToDevice, stm);
        j.out_geno = d_out_geno + (size_t)l * nrun * gstride;
        j.out_E = d_out_E + (size_t)l * nrun;
        j.out_xyz = d_out_xyz ? d_out_xyz + (size_t)l * nrun * cstride * 3 : nullptr;
        j.out_evals = d_out_evals + (size_t)l * nrun;
        j.out_gens = d_out_gens + (size_t)l * nrun;
    }
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("dock alloc: ") + cudaGetErrorString(e));
    CUDA_TRY(cudaMemcpyAsync(d_jobs, jobs.data(), (size_t)nlig * sizeof(DockJob), cudaMemcpyHostToDevice, stm));
    if (best_coords) CUDA_TRY(cudaMemsetAsync(d_out_xyz, 0, (size_t)nlig * nrun * cstride * 12, stm));
    CUDA_TRY(cudaMemsetAsync(d_out_geno, 0, (size_t)nlig * nrun * gstride * 4, stm));

    const size_t smem_ga = cta_smem(maxblob, maxscr, Wga), smem_ls = cta_smem(maxblob, maxscr, Wls);
    CUDA_TRY(cudaFuncSetAttribute(dock_init_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ga));
    CUDA_TRY(cudaFuncSetAttribute(dock_ga_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ga));
    CUDA_TRY(cudaFuncSetAttribute(dock_ls_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ls));
    CUDA_TRY(cudaFuncSetAttribute(dock_final_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ls));

    DockDims dga = dm, dls = dm, dfin = dm, dteam = dm, dgl = dm;
    dgl.upj = (int)((popsz + 127) / 128);                       // thread per individual (dock_ga_lane_kernel)
    dteam.upj = std::max(1, (nrun * dm.n_ls + team_tpc - 1) / team_tpc);     // team_tpc chains per CTA
    if (ls_team && team_tpc == 1) CUDA_TRY(cudaFuncSetAttribute(dock_ls_team_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_team));
    if (ls_team && team_tpc == 4) CUDA_TRY(cudaFuncSetAttribute(dock_ls_team_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_team));
    dga.upj = (int)((popsz + Wga - 1) / Wga);
    dls.upj = std::max(1, (nrun * dm.n_ls + Wls - 1) / Wls);
    dfin.upj = (nrun + Wls - 1) / Wls;
    // lane family: flat group sequence over all jobs (lane_plan)
    LaneDockArgs al{}, as{};
    float* d_lscratch = nullptr;
    int q_tpc = 0, q_nctas = 0;                                 // queue mode of the local-search kernel (0: flat partition)
    size_t q_smem = 0;
    if (ls_lane && dm.n_ls > 0) {
        const size_t T = (size_t)std::max(pl.nctas, g_sm_count) * (kLaneVars[pl.var].W / kLaneVars[pl.var].K) * 32;   // either mode
        cudaError_t e2 = buf.alloc(&d_lscratch, kLaneVars[pl.var].TM ? 16 : T * (size_t)(Gmax + 2 * (Gmax - 1)) * 4);
        if (e2 != cudaSuccess) return fail(e2 == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("dock alloc: ") + cudaGetErrorString(e2));
        al = LaneDockArgs{d_lscratch, Gmax, pl.ng, nlig * jg, jg, pl.slot, pl.nimg, pl.gfloats, 0, nullptr, nullptr};
        // queue mode (on request, see below): tpc teams of jg groups per CTA, as many as fit; needs a ligand for every team of a
        // full wave
        const LaneVar& V = kLaneVars[pl.var];
        const int floats = lane_var_floats(lg, pl.var, true);
        for (int t = std::min(kLaneQueueMaxTeams, (V.W / V.K) / jg); t >= 1 && !q_tpc; --t) {
            const size_t need = kLaneQueueHeader + (size_t)t * pl.slot + (size_t)t * jg * floats * 128;
            const bool cols = !V.TM || 3 * lg.npad <= lane_tmem_columns(t * jg * V.K);
            if (cols && need <= (size_t)g_smem_optin) { q_tpc = t; q_smem = need; }
        }
        if ((long long)nlig < (long long)q_tpc * g_sm_count) q_tpc = 0;     // fewer ligands than teams of a wave: the flat partition spreads them
        {
            double m = 0, v = 0;
            for (double c : cost) m += c;
            m /= nlig;
            for (double c : cost) v += (c - m) * (c - m);
            const double cv = std::sqrt(v / nlig) / m;
            // Measured (profiles/r02_lane_variants.md): the flat partition with the ligands sorted by cost over two or more
            // waves lets the hardware's CTA scheduler do the balancing and beats the queues (whose loop costs the
            // evaluation 6 %) on the bench batch and on configs[2] alike, so the queues run only on request.
            const char* force = std::getenv("ADOCK_LS_QUEUE");              // A/B switch of the profiles: 1 = queues
            (void)cv;
            if (!(force && force[0] == '1')) q_tpc = 0;
        }
        if (q_tpc) {
            q_nctas = std::min(g_sm_count, (nlig + q_tpc - 1) / q_tpc);
            const int nteams = q_nctas * q_tpc;
            // longest processing time first: jobs by decreasing cost, each to the CTA with the least work so far (the warps
            // of an SM share its issue slots) and there to the least loaded team
            std::vector<int> by(nlig);
            std::iota(by.begin(), by.end(), 0);
            std::stable_sort(by.begin(), by.end(), [&](int x, int y) { return cost[jorder[x]] > cost[jorder[y]]; });
            std::vector<double> load(nteams, 0.0), cta_load(q_nctas, 0.0);
            std::vector<std::vector<int>> q(nteams);
            for (int k : by) {
                const int c = (int)(std::min_element(cta_load.begin(), cta_load.end()) - cta_load.begin());
                const int tmin = (int)(std::min_element(load.begin() + c * q_tpc, load.begin() + (c + 1) * q_tpc) - load.begin());
                q[tmin].push_back(k);                           // k = position in jobs[]
                load[tmin] += cost[jorder[k]];
                cta_load[c] += cost[jorder[k]];
            }
            std::vector<int> off(nteams + 1, 0), flat;
            for (int t = 0; t < nteams; ++t) { flat.insert(flat.end(), q[t].begin(), q[t].end()); off[t + 1] = (int)flat.size(); }
            int *d_off = nullptr, *d_q = nullptr;
            e2 = buf.alloc(&d_off, off.size() * 4);
            if (e2 == cudaSuccess) e2 = buf.alloc(&d_q, flat.size() * 4);
            if (e2 == cudaSuccess) e2 = cudaMemcpyAsync(d_off, off.data(), off.size() * 4, cudaMemcpyHostToDevice, stm);
            if (e2 == cudaSuccess) e2 = cudaMemcpyAsync(d_q, flat.data(), flat.size() * 4, cudaMemcpyHostToDevice, stm);
            if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(stm);     // off / flat leave scope
            if (e2 != cudaSuccess) return fail(ADOCK_ECUDA, std::string("dock queue: ") + cudaGetErrorString(e2));
            al.ng = q_tpc * jg; al.nimg = q_tpc; al.tpc = q_tpc; al.q_off = d_off; al.q_job = d_q;
            al.group_floats = floats;
            cudaError_t e4 = cudaSuccess;
            LANE_VARIANT(pl.var, e4 = cudaFuncSetAttribute(dock_ls_lane_queue_kernel<C, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q_smem);
                         if (e4 == cudaSuccess) e4 = cudaFuncSetAttribute(dock_ls_lane_queue_kernel<C, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q_smem))
            CUDA_TRY(e4);
        }
        cudaError_t e3 = cudaSuccess;
        LANE_VARIANT(pl.var, e3 = cudaFuncSetAttribute(dock_ls_lane_kernel<C, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
                     if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(dock_ls_lane_kernel<C, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem))
        CUDA_TRY(e3);
    }
    if (ga_lane) {
        as = LaneDockArgs{nullptr, Gmax, ps.ng, nlig * jgs, jgs, ps.slot, ps.nimg, ps.gfloats};
        cudaError_t e3 = cudaSuccess;
        LANE_VARIANT(ps.var, e3 = cudaFuncSetAttribute(dock_score_lane_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ps.smem))
        CUDA_TRY(e3);
        CUDA_TRY(cudaFuncSetAttribute(dock_ga_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ga));
    }
    auto launch_ls = [&]() {
        const int thr = pl.ng * pl.K * 32;
        const bool sw = p.ls_method == 1;
        if (ls_lane && q_tpc && !sw) { LANE_VARIANT(pl.var, dock_ls_lane_queue_kernel<C, false><<<q_nctas, q_tpc * jg * C::K * 32, q_smem, stm>>>(grids->dev, P, d_jobs, dm, al)) }
        else if (ls_lane && q_tpc) { LANE_VARIANT(pl.var, dock_ls_lane_queue_kernel<C, true><<<q_nctas, q_tpc * jg * C::K * 32, q_smem, stm>>>(grids->dev, P, d_jobs, dm, al)) }
        else if (ls_lane && !sw) { LANE_VARIANT(pl.var, dock_ls_lane_kernel<C, false><<<pl.nctas, thr, pl.smem, stm>>>(grids->dev, P, d_jobs, dm, al)) }
        else if (ls_lane) { LANE_VARIANT(pl.var, dock_ls_lane_kernel<C, true><<<pl.nctas, thr, pl.smem, stm>>>(grids->dev, P, d_jobs, dm, al)) }
        else if (ls_team && team_tpc == 1) dock_ls_team_kernel<1><<<dteam.upj * nlig, kTeamW * 32, smem_team, stm>>>(grids->dev, P, d_jobs, dteam, maxteam);
        else if (ls_team) dock_ls_team_kernel<4><<<dteam.upj * nlig, 4 * kTeamW * 32, smem_team, stm>>>(grids->dev, P, d_jobs, dteam, maxteam);
        else dock_ls_kernel<<<dls.upj * nlig, Wls * 32, smem_ls, stm>>>(grids->dev, P, d_jobs, dls);
    };
    // one GA generation: offspring + their energies (one launch, or two when the scoring runs lane-per-individual)
    auto launch_ga = [&]() {
        if (!ga_lane) {
            dock_ga_kernel<true><<<dga.upj * nlig, Wga * 32, smem_ga, stm>>>(grids->dev, P, d_jobs, dga, nullptr);
            return 1;
        }
        dock_ga_lane_kernel<<<dgl.upj * nlig, 128, 0, stm>>>(P, d_jobs, dgl, nullptr);
        const int thr = ps.ng * ps.K * 32;
        LANE_VARIANT(ps.var, dock_score_lane_kernel<C><<<ps.nctas, thr, ps.smem, stm>>>(grids->dev, P, d_jobs, dm, as))
        return 2;
    };
    dock_init_kernel<<<dga.upj * nlig, Wga * 32, smem_ga, stm>>>(grids->dev, P, d_jobs, dga);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    const bool can_run = (long long)Pn < max_evals && p.max_gens > 0;
    int h_flag = can_run ? 1 : 0;
    const int poll = 8;
    struct EventList {                                  // destroyed on every way out of the function
        std::vector<cudaEvent_t> v;
        ~EventList() { for (cudaEvent_t ev : v) cudaEventDestroy(ev); }
    } prof;
    std::vector<cudaEvent_t>& prof_ev = prof.v;
    for (int g = 0; h_flag && g < p.max_gens; ++g) {
        g_launches += launch_ga() - 1;
        if (dm.n_ls > 0 && p.lsit > 0) {
            if (g_prof) {
                cudaEvent_t a, b;
                CUDA_TRY(cudaEventCreate(&a)); CUDA_TRY(cudaEventCreate(&b));
                CUDA_TRY(cudaEventRecord(a, stm));
                launch_ls();
                CUDA_TRY(cudaEventRecord(b, stm));
                prof_ev.push_back(a); prof_ev.push_back(b);
            } else {
                launch_ls();
            }
        }
        const bool check = ((g + 1) % poll) == 0;
        if (check) CUDA_TRY(cudaMemsetAsync(d_flag, 0, 4, stm));
        dock_commit_kernel<<<nlig, 128, 0, stm>>>(d_jobs, nlig, dm, d_flag);
        g_launches += (dm.n_ls > 0 && p.lsit > 0) ? 3 : 2;
        if (check) {
            CUDA_TRY(cudaMemcpyAsync(&h_flag, d_flag, 4, cudaMemcpyDeviceToHost, stm));
            CUDA_TRY(cudaStreamSynchronize(stm));
        }
    }
    dock_final_kernel<<<dfin.upj * nlig, Wls * 32, smem_ls, stm>>>(grids->dev, P, d_jobs, dfin);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    std::vector<long long> h_evals((size_t)nlig * nrun);
    CUDA_TRY(cudaMemcpyAsync(best_genotypes, d_out_geno, (size_t)nlig * nrun * gstride * 4, cudaMemcpyDeviceToHost, stm));
    CUDA_TRY(cudaMemcpyAsync(best_energies, d_out_E, (size_t)nlig * nrun * 4, cudaMemcpyDeviceToHost, stm));
    if (best_coords) CUDA_TRY(cudaMemcpyAsync(best_coords, d_out_xyz, (size_t)nlig * nrun * cstride * 12, cudaMemcpyDeviceToHost, stm));
    if (evals_used) CUDA_TRY(cudaMemcpyAsync(evals_used, d_out_evals, (size_t)nlig * nrun * 8, cudaMemcpyDeviceToHost, stm));
    if (gens_used) CUDA_TRY(cudaMemcpyAsync(gens_used, d_out_gens, (size_t)nlig * nrun * 4, cudaMemcpyDeviceToHost, stm));
    std::vector<int> h_gens;
    if (g_prof) {
        h_gens.resize((size_t)nlig * nrun);
        CUDA_TRY(cudaMemcpyAsync(h_evals.data(), d_out_evals, (size_t)nlig * nrun * 8, cudaMemcpyDeviceToHost, stm));
        CUDA_TRY(cudaMemcpyAsync(h_gens.data(), d_out_gens, (size_t)nlig * nrun * 4, cudaMemcpyDeviceToHost, stm));
    }
    CUDA_TRY(cudaStreamSynchronize(stm));
    if (g_prof) {
        for (size_t i = 0; i + 1 < prof_ev.size(); i += 2) {
            float ms = 0;
            cudaEventElapsedTime(&ms, prof_ev[i], prof_ev[i + 1]);
            g_ls_ms += ms;
            ++g_ls_launches;
        }
        for (size_t i = 0; i < h_gens.size(); ++i) g_ls_evals += h_evals[i] - Pn - (long long)h_gens[i] * (Pn - 1);
    }
    return ADOCK_OK;
}

extern "C" int adock_dock(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params, int nrun, int pop_size,
                          long long max_evals, unsigned long long seed, float* best_genotypes, float* best_energies,
                          float* best_coords, long long* evals_used, int* gens_used, void* cuda_stream) {
    if (!ligand) return fail(ADOCK_EINVAL, "NULL ligand");
    const adock_ligand* ligs[1] = {ligand};
    return dock_impl(grids, ligs, 1, params, nrun, pop_size, max_evals, &seed, 7 + ligand->tp.R, best_genotypes, best_energies,
                     ligand->tp.N, best_coords, evals_used, gens_used, (cudaStream_t)cuda_stream);
}

extern "C" int adock_dock_many(const adock_grids* grids, const adock_ligand* const* ligands, int nlig, const adock_params* params,
                               int nrun, int pop_size, long long max_evals, const unsigned long long* seeds, int gstride,
                               float* best_genotypes, float* best_energies, int cstride, float* best_coords, long long* evals_used,
                               int* gens_used, void* cuda_stream) {
    return dock_impl(grids, ligands, nlig, params, nrun, pop_size, max_evals, seeds, gstride, best_genotypes, best_energies, cstride,
                     best_coords, evals_used, gens_used, (cudaStream_t)cuda_stream);
}

// =================================================================== screening pipeline (row a7; S8(f) NEXT-3)
// PAPER.md lines 102, 124, 180 and Fig. 1 hide the host-side setup of ligand i+1 behind the docking of ligand i with
// OpenMP threads.  Here the unit is a BATCH of ligands (one launch sequence docks all of them): a prepared batch owns
// its host-only ligand handles, one pinned staging buffer and one device slab holding every image of the batch.
namespace {
struct ScreenBatch {
    std::vector<adock_ligand*> ligs;        // host-only handles, device pointers patched into the slab
    std::vector<int> index;                 // caller's ligand index of each
    unsigned char* pinned = nullptr;
    unsigned char* slab = nullptr;
    size_t bytes = 0;
    cudaEvent_t ready = nullptr;
    int rc = ADOCK_OK;
    std::string err;
    double prep_s = 0;
    void release() {
        for (adock_ligand* l : ligs) adock_free_ligand(l);
        ligs.clear();
        if (pinned) cudaFreeHost(pinned);
        if (slab) cudaFree(slab);
        if (ready) cudaEventDestroy(ready);
        pinned = slab = nullptr; ready = nullptr;
    }
};
inline size_t up128(size_t x) { return (x + 127) & ~(size_t)127; }

// host preprocessing of the batch on `nthr` threads, then one pinned -> device copy of all images on `copy`
void screen_prepare(ScreenBatch& b, int dev, const adock_params* params, int T, const float* coeffs, const float* solpar,
                    const float* vol, const adock_ligand_desc* ligs, int nthr, cudaStream_t copy) {
    const auto t0 = std::chrono::steady_clock::now();
    const int n = (int)b.index.size();
    b.ligs.assign(n, nullptr);
    std::atomic<int> next{0}, bad{-1};
    std::vector<std::string> errs(n);
    std::vector<int> rcs(n, ADOCK_OK);
    auto work = [&]() {
        for (int k = next.fetch_add(1); k < n; k = next.fetch_add(1)) {
            const adock_ligand_desc& d = ligs[b.index[k]];
            rcs[k] = adock_load_ligand(nullptr, params, d.N, d.xyz, d.type, d.charge, d.nbonds, d.bonds, d.R, d.rot_bonds, d.root_atom,
                                       T, coeffs, solpar, vol, &b.ligs[k]);
            if (rcs[k] != ADOCK_OK) { errs[k] = g_err; int exp = -1; bad.compare_exchange_strong(exp, k); }
        }
    };
    std::vector<std::thread> pool;
    for (int t = 1; t < nthr; ++t) pool.emplace_back(work);
    work();
    for (auto& th : pool) th.join();
    if (bad.load() >= 0) {
        const int k = bad.load();
        b.rc = rcs[k]; b.err = "ligand " + std::to_string(b.index[k]) + ": " + errs[k];
        return;
    }
    size_t off = 0;
    std::vector<size_t> o_blob(n), o_ext(n), o_lane(n);
    for (int k = 0; k < n; ++k) {
        const adock_ligand* l = b.ligs[k];
        o_blob[k] = off; off += up128((size_t)l->blob_bytes);
        o_ext[k] = off; off += up128(l->tp.ext_of_int.size() * sizeof(int));
        o_lane[k] = off; off += up128((size_t)l->lane_bytes);
    }
    b.bytes = off;
    cudaError_t e = cudaSetDevice(dev);
    if (e == cudaSuccess) e = cudaMallocHost(&b.pinned, off);
    if (e == cudaSuccess) e = cudaMalloc(&b.slab, off);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&b.ready, cudaEventDisableTiming);
    if (e == cudaSuccess) {
        for (int k = 0; k < n; ++k) {
            adock_ligand* l = b.ligs[k];
            std::memcpy(b.pinned + o_blob[k], l->tp.blob.data(), (size_t)l->blob_bytes);
            std::memcpy(b.pinned + o_ext[k], l->tp.ext_of_int.data(), l->tp.ext_of_int.size() * sizeof(int));
            std::memcpy(b.pinned + o_lane[k], l->lane.blob.data(), (size_t)l->lane_bytes);
            l->d_blob = b.slab + o_blob[k];
            l->d_ext_of_int = reinterpret_cast<int*>(b.slab + o_ext[k]);
            l->d_lane = b.slab + o_lane[k];
            l->owns_dev = false;
        }
        e = cudaMemcpyAsync(b.slab, b.pinned, off, cudaMemcpyHostToDevice, copy);
    }
    if (e == cudaSuccess) e = cudaEventRecord(b.ready, copy);
    if (e != cudaSuccess) { b.rc = e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA; b.err = std::string("screen upload: ") + cudaGetErrorString(e); }
    b.prep_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
}
}  // namespace

extern "C" int adock_screen(const adock_grids* grids, const adock_params* params, int T, const float* pair_coeffs, const float* solpar,
                            const float* vol, int nlig, const adock_ligand_desc* ligs, int nrun, int pop_size, long long max_evals,
                            const unsigned long long* seeds, int batch, int host_threads, int gstride, float* best_genotypes,
                            float* best_energies, long long* evals_used, adock_screen_stats* stats, void* cuda_stream) {
    if (stats) *stats = adock_screen_stats{};
    if (!grids || !pair_coeffs || !solpar || !vol || !best_genotypes || !best_energies) return fail(ADOCK_EINVAL, "NULL argument");
    if (nlig < 0 || batch < 0 || host_threads < 1 || nrun < 1 || pop_size < 2) return fail(ADOCK_EINVAL, "bad screening dimensions");
    if (nlig == 0) return ADOCK_OK;
    if (!ligs || !seeds) return fail(ADOCK_EINVAL, "NULL argument");
    int maxG = 7;
    for (int i = 0; i < nlig; ++i) {
        if (ligs[i].N < 1 || ligs[i].R < 0) return fail(ADOCK_EINVAL, "ligand " + std::to_string(i) + ": bad shape");
        maxG = std::max(maxG, 7 + ligs[i].R);
    }
    if (gstride < maxG) return fail(ADOCK_EINVAL, "output stride too small");
    int rc = device_props();
    if (rc) return rc;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    const auto t_start = std::chrono::steady_clock::now();
    // batches of similar size: stable sort by atom count (largest first)
    std::vector<int> order(nlig);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return ligs[a].N > ligs[b].N; });
    // batch boundaries: fixed length, or (batch == 0) as many ligands as fill ONE wave of the lane-per-individual local-search
    // kernel at the estimated geometry of the batch's largest ligand (first of the batch): 148 SMs x groups per CTA
    std::vector<int> bstart{0};
    if (batch > 0) {
        for (int i = batch; i < nlig; i += batch) bstart.push_back(i);
    } else {
        adock_params pp;
        rc = check_params(params, nullptr, pp);
        if (rc) return rc;
        const int jg = std::max(1, (nrun * n_ls_of(pp, pop_size) + 31) / 32);
        // geometry of the largest ligand (first in the order), estimated from its descriptor: image ~ 7.6 N^2 bytes (two
        // slots), 6 accumulator floats per fragment.  Batch length = two ligands per team of the local-search kernel at that
        // geometry (its work queues balance them by cost; measured on configs[2]: profiles/r02_lane_variants.md), equalised
        // over the batches so that no small tail batch falls back to the warp-per-individual kernels.
        const adock_ligand_desc& d = ligs[order[0]];
        const int npad = (d.N + kLaneBI - 1) / kLaneBI * kLaneBI;
        LaneGeom g{2 * (8 * d.N * d.N + 512), npad, 6 * (d.R + 1), d.R};
        const int ng = std::max(1, lane_plan(g, 1 << 20, jg, true).ng);      // groups per CTA of the variant the docking will pick
        const int target = std::max(1, 2 * g_sm_count * ng / jg);
        const int nbat = (nlig + target - 1) / target;
        for (int b = 1; b < nbat; ++b) bstart.push_back((int)((long long)nlig * b / nbat));
    }
    bstart.push_back(nlig);
    const int nb = (int)bstart.size() - 1;
    cudaStream_t stm = (cudaStream_t)cuda_stream, copy = nullptr;
    CUDA_TRY(cudaStreamCreateWithFlags(&copy, cudaStreamNonBlocking));
    ScreenBatch slot[2];
    auto fill = [&](ScreenBatch& b, int bi) {
        b.index.assign(order.begin() + bstart[bi], order.begin() + bstart[bi + 1]);
        screen_prepare(b, dev, params, T, pair_coeffs, solpar, vol, ligs, host_threads, copy);
    };
    double dock_s = 0, prep_s = 0, exposed_s = 0;
    std::string err;
    std::thread producer;
    {
        const auto t0 = std::chrono::steady_clock::now();
        fill(slot[0], 0);
        exposed_s += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    }
    std::vector<float> bg, bE;
    std::vector<long long> bev;
    std::vector<unsigned long long> bseed;
    for (int bi = 0; bi < nb && rc == ADOCK_OK; ++bi) {
        ScreenBatch& cur = slot[bi & 1];
        if (bi + 1 < nb) producer = std::thread(fill, std::ref(slot[(bi + 1) & 1]), bi + 1);     // overlaps the docking below
        if (cur.rc != ADOCK_OK) { rc = cur.rc; err = cur.err; }
        if (rc == ADOCK_OK) {
            const int n = (int)cur.index.size();
            prep_s += cur.prep_s;
            cudaError_t e = cudaStreamWaitEvent(stm, cur.ready, 0);
            if (e != cudaSuccess) { rc = ADOCK_ECUDA; err = std::string("screen: ") + cudaGetErrorString(e); }
            if (rc == ADOCK_OK) {
                bg.assign((size_t)n * nrun * gstride, 0.f); bE.assign((size_t)n * nrun, 0.f); bev.assign((size_t)n * nrun, 0); bseed.resize(n);
                for (int k = 0; k < n; ++k) bseed[k] = seeds[cur.index[k]];
                const auto t0 = std::chrono::steady_clock::now();
                rc = dock_impl(grids, cur.ligs.data(), n, params, nrun, pop_size, max_evals, bseed.data(), gstride, bg.data(), bE.data(), 0,
                               nullptr, bev.data(), nullptr, stm);
                dock_s += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
                if (rc != ADOCK_OK) err = g_err;
                for (int k = 0; k < n && rc == ADOCK_OK; ++k) {
                    const size_t dst = (size_t)cur.index[k];
                    std::memcpy(best_genotypes + dst * nrun * gstride, bg.data() + (size_t)k * nrun * gstride, (size_t)nrun * gstride * 4);
                    std::memcpy(best_energies + dst * nrun, bE.data() + (size_t)k * nrun, (size_t)nrun * 4);
                    if (evals_used) std::memcpy(evals_used + dst * nrun, bev.data() + (size_t)k * nrun, (size_t)nrun * 8);
                }
            }
        }
        if (producer.joinable()) {
            const auto t0 = std::chrono::steady_clock::now();
            producer.join();
            exposed_s += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
        }
        cur.release();
    }
    if (producer.joinable()) producer.join();
    slot[0].release(); slot[1].release();
    cudaStreamDestroy(copy);
    if (stats) {
        stats->wall_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
        stats->dock_s = dock_s; stats->prep_s = prep_s; stats->exposed_s = exposed_s; stats->batches = nb; stats->host_threads = host_threads;
    }
    if (rc != ADOCK_OK) return fail(rc, err);
    return ADOCK_OK;
}

// =================================================================== pose post-processing (R13)
// one warp per ordered pair (a, b), b in [0, n]: b == n is the reference pose
__global__ void __launch_bounds__(256) pose_rmsd_kernel(const float* __restrict__ x, const float* __restrict__ ref, int n, int N,
                                                        float* __restrict__ out_ref, float* __restrict__ out_pair) {
    const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= (long long)n * (n + 1)) return;
    const int a = (int)(w / (n + 1)), b = (int)(w % (n + 1));
    if (b == n ? !out_ref : (!out_pair || b < a)) return;
    const float* pa = x + (size_t)a * N * 3;
    const float* pb = b == n ? ref : x + (size_t)b * N * 3;
    float s = 0.f;
    for (int i = lane; i < 3 * N; i += 32) { const float d = pa[i] - pb[i]; s = fmaf(d, d, s); }
    s = warp_sum(s);
    if (lane == 0) {
        const float r = sqrtf(s / (float)N);
        if (b == n) out_ref[a] = r;
        else { out_pair[(size_t)a * n + b] = r; out_pair[(size_t)b * n + a] = r; }
    }
}

extern "C" int adock_pose_rmsd(int n, int N, const float* coords, const float* ref, float* rmsd_ref, float* rmsd_pair,
                               const float* energies, float tol, int* cluster, int* nclusters, void* cuda_stream) {
    if (n < 0 || N < 1) return fail(ADOCK_EINVAL, "bad pose dimensions");
    if (n > 32768) return fail(ADOCK_ELIMIT, "more than 32768 poses");
    if (nclusters) *nclusters = 0;
    if (n == 0) return ADOCK_OK;
    if (!coords || (rmsd_ref && !ref) || (cluster && (!energies || !(tol > 0) || !nclusters))) return fail(ADOCK_EINVAL, "NULL argument");
    for (size_t i = 0; i < (size_t)n * N * 3; ++i) if (!std::isfinite(coords[i])) return fail(ADOCK_EINVAL, "non-finite coordinate");
    cudaStream_t stm = (cudaStream_t)cuda_stream;
    const bool want_pair = rmsd_pair || cluster;
    DevBuf buf;
    float *d_x = nullptr, *d_ref = nullptr, *d_or = nullptr, *d_op = nullptr;
    cudaError_t e = buf.alloc(&d_x, (size_t)n * N * 12);
    if (e == cudaSuccess && rmsd_ref) e = buf.alloc(&d_ref, (size_t)N * 12);
    if (e == cudaSuccess && rmsd_ref) e = buf.alloc(&d_or, (size_t)n * 4);
    if (e == cudaSuccess && want_pair) e = buf.alloc(&d_op, (size_t)n * n * 4);
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ADOCK_ENOMEM : ADOCK_ECUDA, std::string("rmsd alloc: ") + cudaGetErrorString(e));
    CUDA_TRY(cudaMemcpyAsync(d_x, coords, (size_t)n * N * 12, cudaMemcpyHostToDevice, stm));
    if (rmsd_ref) CUDA_TRY(cudaMemcpyAsync(d_ref, ref, (size_t)N * 12, cudaMemcpyHostToDevice, stm));
    const long long warps = (long long)n * (n + 1);
    pose_rmsd_kernel<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, stm>>>(d_x, d_ref, n, N, d_or, d_op);
    ++g_launches;
    CUDA_TRY(cudaGetLastError());
    std::vector<float> pair;
    if (rmsd_ref) CUDA_TRY(cudaMemcpyAsync(rmsd_ref, d_or, (size_t)n * 4, cudaMemcpyDeviceToHost, stm));
    if (want_pair) {
        pair.resize((size_t)n * n);
        CUDA_TRY(cudaMemcpyAsync(pair.data(), d_op, (size_t)n * n * 4, cudaMemcpyDeviceToHost, stm));
    }
    CUDA_TRY(cudaStreamSynchronize(stm));
    if (rmsd_pair) std::memcpy(rmsd_pair, pair.data(), (size_t)n * n * 4);
    if (cluster) {
        std::vector<int> order(n), seeds;
        std::iota(order.begin(), order.end(), 0);
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return energies[a] < energies[b]; });
        for (int k : order) {
            int c = -1;
            for (size_t s = 0; s < seeds.size() && c < 0; ++s)
                if (pair[(size_t)k * n + seeds[s]] <= tol) c = (int)s;
            if (c < 0) { c = (int)seeds.size(); seeds.push_back(k); }
            cluster[k] = c;
        }
        *nclusters = (int)seeds.size();
    }
    return ADOCK_OK;
}

// =================================================================== GA test hook (R9): one generation, no scoring
extern "C" int adock_ga_generation(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params, int nrun, int Pn,
                                   int generation, unsigned long long seed, const float* d_pop, const float* d_energies,
                                   float* d_newpop, int* d_decisions, int* d_ls_picks, int* n_ls, void* cuda_stream) {
    if (!grids || !ligand || !d_newpop) return fail(ADOCK_EINVAL, "NULL argument");
    if (nrun < 1 || Pn < 2 || generation < 0 || (generation > 0 && (!d_pop || !d_energies))) return fail(ADOCK_EINVAL, "bad GA arguments");
    adock_params p;
    int rc = check_params(params, ligand, p);
    if (rc) return rc;
    rc = device_props();
    if (rc) return rc;
    cudaStream_t stm = (cudaStream_t)cuda_stream;
    const int W = fit_warps(ligand->blob_bytes, ligand->scratch_floats, 8);
    if (!W) return fail(ADOCK_ELIMIT, "ligand does not fit in shared memory");
    const size_t smem = cta_smem(ligand->blob_bytes, ligand->scratch_floats, W);
    ParDev P = make_pardev(p);
    P.k_wall_h = p.k_wall * grids->dev.h;
    const size_t popsz = (size_t)nrun * Pn;
    const int Gn = 7 + ligand->tp.R;
    DevBuf buf;
    DockJob j{};
    j.blob = ligand->d_blob; j.ext_of_int = ligand->d_ext_of_int; j.blob_bytes = ligand->blob_bytes;
    j.Gn = Gn; j.N = ligand->tp.N; j.R = ligand->tp.R; j.seed = seed;
    DockJob* d_job = nullptr;
    cudaError_t e = buf.alloc(&j.pop, 2 * popsz * Gn * 4);
    if (e == cudaSuccess) e = buf.alloc(&j.E, 2 * popsz * 4);
    if (e == cudaSuccess) e = buf.alloc(&j.st, (size_t)nrun * sizeof(RunState));
    if (e == cudaSuccess) e = buf.alloc(&j.picks, popsz * 4);
    if (e == cudaSuccess) e = buf.alloc(&j.fy, popsz * 4);
    if (e == cudaSuccess) e = buf.alloc(&d_job, sizeof(DockJob));
    if (e != cudaSuccess) return fail(ADOCK_ENOMEM, std::string("ga alloc: ") + cudaGetErrorString(e));
    DockDims dm{};
    dm.nrun = nrun; dm.P = Pn; dm.n_ls = n_ls_of(p, Pn); dm.max_evals = (1ll << 60); dm.max_gens = 1 << 30;
    dm.upj = (int)((popsz + W - 1) / W);
    if (n_ls) *n_ls = dm.n_ls;
    CUDA_TRY(cudaMemcpyAsync(d_job, &j, sizeof(DockJob), cudaMemcpyHostToDevice, stm));
    if (generation == 0) {
        CUDA_TRY(cudaFuncSetAttribute(dock_init_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        dock_init_kernel<<<dm.upj, W * 32, smem, stm>>>(grids->dev, P, d_job, dm);
        ++g_launches;
        CUDA_TRY(cudaMemcpyAsync(d_newpop, j.pop, popsz * Gn * 4, cudaMemcpyDeviceToDevice, stm));
    } else {
        std::vector<RunState> st(nrun);
        for (auto& s : st) { s.evals = 0; s.gen = generation - 1; s.cur = 0; s.active = 1; s.ls_acc = 0; s.pad[0] = s.pad[1] = 0; }
        CUDA_TRY(cudaMemcpyAsync(j.st, st.data(), nrun * sizeof(RunState), cudaMemcpyHostToDevice, stm));
        CUDA_TRY(cudaMemcpyAsync(j.pop, d_pop, popsz * Gn * 4, cudaMemcpyDeviceToDevice, stm));
        CUDA_TRY(cudaMemcpyAsync(j.E, d_energies, popsz * 4, cudaMemcpyDeviceToDevice, stm));
        if (g_path == 2) {                              // lane family: the thread-per-individual kernel of the batched dockings
            DockDims dl = dm;
            dl.upj = (int)((popsz + 127) / 128);
            dock_ga_lane_kernel<<<dl.upj, 128, 0, stm>>>(P, d_job, dl, d_decisions);
        } else {
            CUDA_TRY(cudaFuncSetAttribute(dock_ga_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            dock_ga_kernel<false><<<dm.upj, W * 32, smem, stm>>>(grids->dev, P, d_job, dm, d_decisions);
        }
        ++g_launches;
        CUDA_TRY(cudaMemcpyAsync(d_newpop, j.pop + popsz * Gn, popsz * Gn * 4, cudaMemcpyDeviceToDevice, stm));
        if (d_ls_picks) CUDA_TRY(cudaMemcpyAsync(d_ls_picks, j.picks, popsz * 4, cudaMemcpyDeviceToDevice, stm));
    }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(stm));
    return ADOCK_OK;
}

// =================================================================== measurement utility: the ALU roofline's peak
// The hot path is bound by plain FP32 arithmetic, for which MEASURED_PEAKS.json has no figure.
// This kernel measures it where the benchmark runs: 8 independent chains of fma.rn.f32x2 per thread, 16 warps per SM,
// one CTA per SM; FLOP = 2 (FMA) x 2 (lanes of the packed operand) per instruction and thread.
__global__ void __launch_bounds__(512) alu_peak_kernel(float* out, int iters, float seed) {
    f2 p[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) p[i] = pk(seed + i, seed - i);
    const f2 a = pk(0.999f, 1.001f), b = pk(1e-3f, -1e-3f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(p[i].v) : "l"(p[i].v), "l"(a.v), "l"(b.v));
        }
    }
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += hsum(p[i]);
    if (acc == 12345.678f) out[0] = acc;
}

extern "C" int adock_alu_peak(double* tflops, double* fma_lanes_per_clk_sm, void* cuda_stream) {
    int rc = device_props();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, khz = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    float* d = nullptr;
    CUDA_TRY(cudaMalloc(&d, 4));
    const int iters = 20000, warps = 16;
    cudaEvent_t a = nullptr, b = nullptr;
    cudaError_t e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    float best = 1e30f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {         // first launch = warm-up; best of the other three
        e = cudaEventRecord(a, st);
        alu_peak_kernel<<<g_sm_count, warps * 32, 0, st>>>(d, iters, 1.0f);
        ++g_launches;
        if (e == cudaSuccess) e = cudaEventRecord(b, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(b);
        float ms = 0;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
        if (rep > 0 && ms < best) best = ms;
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(d);
    if (e != cudaSuccess) return fail(ADOCK_ECUDA, std::string("alu_peak: ") + cudaGetErrorString(e));
    const double lanes = (double)g_sm_count * warps * 32 * iters * 4 * 8 * 2.0;       // FMA lanes executed
    if (tflops) *tflops = 2.0 * lanes / (best * 1e-3) / 1e12;
    if (fma_lanes_per_clk_sm) *fma_lanes_per_clk_sm = lanes / (best * 1e-3 * khz * 1e3) / g_sm_count;
    return ADOCK_OK;
}

// =================================================================== tensor memory as per-lane scratch: the measurement
// The TM variants of the lane kernels keep atom positions in tensor memory (lane.cuh).  This probe is the evidence that the
// access pattern is sound and what it costs (profiles/r02_tmem_scratch.md): every warp of a CTA of `warps` warps writes a
// pattern into its slice with tcgen05.st.32x32b and reads it back with .x1 / .x2 / .x4 loads at warp-uniform dynamic
// columns (mode 0: mismatches counted); a pointer chase gives the dependent-load latency (mode 1: tensor memory, mode 3:
// shared memory), 8 independent 64-bit loads per wait the throughput (mode 2: tcgen05.ld.x2, mode 4: LDS.64).
template <int mode>
__global__ void __launch_bounds__(512, 1) tmem_probe_kernel(int iters, int* errors, long long* cycles, float* sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    const uint32_t tmem = lane_tmem_open<true>(smem);
    const int per = lane_tmem_columns(W);
    const uint32_t mine = tmem + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * per);
    float* sm = reinterpret_cast<float*>(smem + 16) + (size_t)warp * 128 * 32 + lane;        // 128 columns per lane
    int err = 0;
    long long t0 = 0, t1 = 0;
    float acc = 0.f;
    if (mode == 0) {
        for (int c = 0; c < per; ++c) tm_st1(mine + c, (float)(warp * 4099 + lane * 67 + c));
        tm_wait_st();
        for (int c = per - 1; c >= 0; --c) {
            float v, d0 = 0.f, d1 = 0.f;
            tm_ld1(mine + c, v);
            tm_wait_ld(v, d0, d1);
            if (v != (float)(warp * 4099 + lane * 67 + c)) ++err;
        }
        for (int m = 0; 6 * m + 5 < per; ++m) {             // the position layout: .x4 at column 6m, .x2 at 6m + 4
            float a, b, c, d, e, f;
            tm_ld4(mine + 6 * m, a, b, c, d);
            tm_ld2(mine + 6 * m + 4, e, f);
            tm_wait_ld(a, b, c, d, e, f);
            const float base = (float)(warp * 4099 + lane * 67 + 6 * m);
            if (a != base || b != base + 1 || c != base + 2 || d != base + 3 || e != base + 4 || f != base + 5) ++err;
        }
    } else if (mode == 1 || mode == 3) {
        for (int c = 0; c < 128; ++c) {
            const float nxt = __int_as_float((c * 37 + 11) & 127);        // the next column, as raw bits (no conversion in the chase)
            if (mode == 1) tm_st1(mine + c, nxt); else sm[c * 32] = nxt;
        }
        tm_wait_st();
        __syncwarp();
        int c = 0;
        t0 = clock64();
        for (int i = 0; i < iters; ++i) {
            float v, d0 = 0.f, d1 = 0.f;
            if (mode == 1) { tm_ld1(mine + c, v); tm_wait_ld(v, d0, d1); } else v = sm[c * 32];
            c = __float_as_int(v);
        }
        t1 = clock64();
        acc = (float)c;
    } else {
        for (int c = 0; c < 128; ++c) { tm_st1(mine + c, 1.0f + c); sm[c * 32] = 1.0f + c; }
        tm_wait_st();
        __syncwarp();
        t0 = clock64();
        for (int i = 0; i < iters; ++i) {
            float v[16];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int c = ((i + k * 6) & 63) * 2;
                if (mode == 2) tm_ld2(mine + c, v[2 * k], v[2 * k + 1]);
                else { const float2 q = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(smem + 16) + ((size_t)warp * 64 + (c >> 1)) * 64 + 2 * lane); v[2 * k] = q.x; v[2 * k + 1] = q.y; }
            }
            if (mode == 2) { tm_wait_ld(v[0], v[1], v[2], v[3], v[4], v[5], v[6], v[7], v[8], v[9], v[10], v[11]); tm_wait_ld(v[12], v[13], v[14]); }
#pragma unroll
            for (int k = 0; k < 16; ++k) acc += v[k];
        }
        t1 = clock64();
    }
    if (err) atomicAdd(errors, err);
    if (lane == 0) cycles[blockIdx.x * W + warp] = t1 - t0;
    sink[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    lane_tmem_close<true>(tmem);
}

extern "C" int adock_tmem_probe(int warps, int mode, int iters, int* errors, double* cycles_per_iteration, void* cuda_stream) {
    if (warps < 1 || warps > 12 || mode < 0 || mode > 4 || iters < 1) return fail(ADOCK_EINVAL, "tmem probe: warps 1..12, mode 0..4, iters >= 1");
    int rc = device_props();
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t smem = 16 + (size_t)warps * 128 * 32 * 4;
    int* d_err = nullptr; long long* d_cyc = nullptr; float* d_sink = nullptr;
    cudaError_t e = cudaMalloc(&d_err, 4);
    if (e == cudaSuccess) e = cudaMalloc(&d_cyc, (size_t)g_sm_count * warps * 8);
    if (e == cudaSuccess) e = cudaMalloc(&d_sink, (size_t)g_sm_count * warps * 32 * 4);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_err, 0, 4, st);
    auto kern = mode == 0 ? tmem_probe_kernel<0> : mode == 1 ? tmem_probe_kernel<1> : mode == 2 ? tmem_probe_kernel<2> : mode == 3 ? tmem_probe_kernel<3> : tmem_probe_kernel<4>;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    std::vector<long long> cyc((size_t)g_sm_count * warps);
    int h_err = 0;
    if (e == cudaSuccess) {
        kern<<<g_sm_count, warps * 32, smem, st>>>(iters, d_err, d_cyc, d_sink);
        ++g_launches;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h_err, d_err, 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(cyc.data(), d_cyc, cyc.size() * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_err); cudaFree(d_cyc); cudaFree(d_sink);
    if (e != cudaSuccess) return fail(ADOCK_ECUDA, std::string("tmem probe: ") + cudaGetErrorString(e));
    double mean = 0;
    for (long long c : cyc) mean += (double)c;
    if (errors) *errors = h_err;
    if (cycles_per_iteration) *cycles_per_iteration = mean / (double)cyc.size() / iters;
    return ADOCK_OK;
}
