/* adock.h -- C ABI of the B200-native (sm_100a) hot path of AutoDock-GPU-style LGA docking.
 *
 * Method: arxiv 2007.03678.  The paper names the computation -- AutoDock4 energy function
 * (line 58), precomputed affinity / electrostatic / desolvation grid maps (line 116), Lamarckian GA with
 * ADADELTA local search and `nrun` independent runs (lines 58, 64), maps loaded once and reused across
 * ligands (lines 100-106) -- but prints no formulas; the exact arithmetic is fixed by the readings
 * R1..R10 in DESIGN.md, which this header cites.
 *
 * Conventions
 *   - Every function returns ADOCK_OK (0) or a negative error code; adock_last_error() returns a
 *     thread-local description of the last failure on the calling thread.
 *   - "host" / "device" on each pointer says where the memory must live.  The caller owns every buffer
 *     it passes; the library owns handles until the matching adock_free_*.
 *   - cuda_stream arguments are a cudaStream_t passed as void* (NULL = default stream).
 *   - All work runs in this library's CUDA kernels.  There is no CPU fallback and no other backend:
 *     without a CUDA device every compute entry point fails with ADOCK_ECUDA.
 *
 * Genotype (R1): float[7+R] = t_x,t_y,t_z (Angstrom, grid frame), q_w,q_x,q_y,q_z (any non-zero
 *   quaternion, normalised on use), tau_1..tau_R (radians, relative to the input conformation, in the
 *   order the rotatable bonds were passed to adock_load_ligand).
 * Gradient (R1,R6): float[6+R] = dE/dt (3, kcal/mol/A), dE/domega (3, kcal/mol/rad; omega = rotation
 *   vector of a left-multiplied infinitesimal rotation about the pivot, q <- exp(omega/2) (x) q),
 *   dE/dtau (R, kcal/mol/rad).
 */
#ifndef ADOCK_H
#define ADOCK_H

#ifdef __cplusplus
extern "C" {
#endif

#define ADOCK_OK 0
#define ADOCK_EINVAL (-1) /* bad shape / index / NULL / non-finite input / params mismatch */
#define ADOCK_ENOMEM (-2) /* host or device allocation failed */
#define ADOCK_ECUDA (-3)  /* CUDA runtime error (text in adock_last_error) or no device */
#define ADOCK_ELIMIT (-4) /* N > 256, R > 64, M > 16, the ligand does not fit in shared memory, or a batch beyond a stated maximum */

#define ADOCK_MAX_ATOMS 256
#define ADOCK_MAX_TORSIONS 64
#define ADOCK_MAX_MAPS 16

typedef struct adock_grids adock_grids;   /* opaque, device resident, immutable, shareable across streams/ligands */
typedef struct adock_ligand adock_ligand; /* opaque, preprocessed topology on host and device, immutable */

/* Every tunable constant of the method (R4,R5,R7,R9).  Force-field fields (first ten) are
 * baked into a ligand at adock_load_ligand; later calls must pass the same values (else ADOCK_EINVAL). */
typedef struct adock_params {
    float elec_scale;  /* W_el * 332.06363 (R5) */
    float diel_A, diel_B, diel_k, diel_lambda; /* eps(r) = A + B/(1 + k exp(-lambda B r)) (R5); k > 0 */
    float w_desolv;    /* W_ds (R5) */
    float ds_sigma;    /* sigma of the desolvation Gaussian, Angstrom (R5) */
    float qasp;        /* S_i = solpar[type_i] + qasp*|q_i| (R5) */
    float r_min;       /* pair distance floor, Angstrom; no force below it (R5) */
    float k_wall;      /* out-of-box linear wall, kcal/mol/Angstrom (R4) */
    float ad_rho, ad_eps; /* ADADELTA decay and epsilon (R7) */
    float lsrat;       /* fraction of the population refined per generation (R9) */
    float tourn_prob, xover_rate, mut_rate; /* GA probabilities (R9) */
    float dmov, dang;  /* mutation amplitudes: Angstrom, radians (R9) */
    int lsit;          /* local-search iterations: ADADELTA 1 eval each (R7); Solis-Wets 1 or 2 evals each (R11) */
    int max_gens;      /* generation cap (R9) */
    /* Local-search method ("Solis-Wets" or "ADADELTA"): 0 = ADADELTA (R7),
     * 1 = Solis-Wets (R11; Solis & Wets 1981 rule, gradient-free). */
    int ls_method;
    int sw_max_succ, sw_max_fail; /* R11: consecutive successes / failures that expand / contract the step scale */
    /* Autostop (R12): when non-zero a run ends after generation g >= as_window once the
     * std-dev of its best energy over the last as_window (1..64) generations is < as_tol (kcal/mol). */
    int autostop, as_window;
    float sw_rho0, sw_rho_lb;       /* R11: initial step scale; the search ends when the scale falls below sw_rho_lb */
    float sw_expand, sw_contract;   /* R11: scale factors (2, 0.5) */
    float sw_bias_keep, sw_bias_gain, sw_bias_decay; /* R11: b <- keep b +- gain delta on success, decay b on failure */
    float as_tol;
} adock_params;

/* Fills *out with the defaults listed in DESIGN.md. */
int adock_default_params(adock_params* out);

/* Grid maps (R4).  host_maps: host, [M][nz][ny][nx] float32, M = T+2:
 * maps 0..T-1 per-atom-type affinity, map T electrostatic potential (multiplied by q_i at lookup), map
 * T+1 desolvation (multiplied by |q_i|).  spacing > 0 in Angstrom; origin: host, xyz of node (0,0,0).
 * The maps are copied and re-laid-out on the device (caller keeps host_maps); node values must be finite. */
int adock_load_grids(const float* host_maps, int M, int nx, int ny, int nz, float spacing, const float origin[3],
                     adock_grids** out);
void adock_free_grids(adock_grids* g);

/* Ligand (R2).  All arrays host.  xyz [N][3] input conformation in the grid frame; type [N] in [0,T);
 * charge [N]; bonds [nbonds][2]; rot_bonds [R][2] (either orientation; a ring bond is ADOCK_EINVAL);
 * root_atom fixes the root fragment; pair_coeffs [T][T][4] = c12, cA, expA (6 or 10), unused -- already
 * weighted; solpar [T], vol [T].  T+2 must be <= grids' M.  params NULL = defaults.
 * grids may be NULL: the handle then carries only the host-side structure (accessors below work, no
 * device memory is touched, compute entry points reject it with ADOCK_EINVAL). */
int adock_load_ligand(const adock_grids* grids, const adock_params* params, int N, const float* xyz, const int* type,
                      const float* charge, int nbonds, const int* bonds, int R, const int* rot_bonds, int root_atom, int T,
                      const float* pair_coeffs, const float* solpar, const float* vol, adock_ligand** out);
void adock_free_ligand(adock_ligand* l);

/* Integer structure of a loaded ligand, canonical order (R2), for bit-exact checks.  Returned pointers
 * are host memory owned by the handle.  pairs [npairs][2] lexicographic (i<j); tor_order [R] deepest first;
 * moved [R][N] 0/1; rot [R][2] oriented (a_k root side, b_k moves); pivot [3]. */
int adock_ligand_pairs(const adock_ligand* l, int* npairs, const int** ij);
int adock_ligand_tree(const adock_ligand* l, const int** tor_order, const unsigned char** moved, const int** rot,
                      const float** pivot);

/* The ligand image the kernels stage into shared memory (host copy, owned by the handle): header,
 * atoms renumbered fragment-contiguously, fragment tree, and the pair list packed into warp rounds of 32
 * slots in which no atom occurs twice as i or twice as j (layout: csrc/topology.hpp).  int_of_ext [N]
 * maps caller atom index -> internal index. */
int adock_ligand_image(const adock_ligand* l, int* bytes, const unsigned char** image, const int** int_of_ext);

/* The ligand image of the lane-per-individual kernels (host copy, owned by the handle): atoms in fragment
 * DFS preorder, fragment tree, and the pair list cut into 4-row x 2-column register tiles with one 32-byte coefficient
 * record per row (layout: csrc/lane_image.hpp).  pos_of_ext [N] maps caller atom index -> position in that order. */
int adock_ligand_lane_image(const adock_ligand* l, int* bytes, const unsigned char** image, const int** pos_of_ext);

/* Kernel family used by the compute entry points of this process: 0 = chosen by problem
 * size (default), 1 = one warp per individual, 2 = one lane per individual with K = 1, 2 or 4 warps sharing the
 * work of each group of 32 individuals (variant chosen by size; 21, 22, 24 force K = 1, 2, 4 with the atom positions in
 * shared memory; 41, 42, 43 force K = 1 with the atom positions in tensor memory and at most 8, 12, 16 warps per SM; a
 * forced variant whose per-lane state does not fit for a ligand makes the compute calls return ADOCK_ELIMIT).  All of them compute
 * the same function (R3-R7) and pass the same parity tests; they differ in summation order only.
 * 3 = the ADADELTA chains of adock_dock / adock_dock_many each run on a team (one CTA of 4 warps per individual,
 * threads over atoms and pairs), chosen by size when a launch holds too few chains to give every scheduler a warp
 * (a single ligand); adock_local_search then runs the same team code on its array of starts (if the ligand fits one
 * team per CTA); every other entry point behaves as with 1. */
int adock_set_path(int path);
/* Family (1, 2 or 3) the local search of the last adock_dock / adock_dock_many on this thread ran in; 0 = none yet. */
int adock_last_dock_path(void);

/* Batched scoring (R3-R6): for each of n genotypes build the pose, interpolate the maps, sum the
 * intramolecular pair terms and back-propagate.  d_genotypes: device [n][gstride], gstride >= 7+R.
 * d_energies: device [n].  d_energy_terms: device [n][2] = (intermolecular, intramolecular) or NULL.
 * d_gradients: device [n][dstride], dstride >= 6+R, or NULL for energy only.  A row with |q| < 1e-12
 * gets NaN energy and gradient.  Asynchronous on cuda_stream. */
int adock_score_batch(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                      const float* d_genotypes, int n, int gstride, float* d_energies, float* d_energy_terms,
                      float* d_gradients, int dstride, void* cuda_stream);

/* Same computation with HOST buffers: copies genotypes in, results out (synchronous). */
int adock_score_batch_host(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                           const float* h_genotypes, int n, int gstride, float* h_energies, float* h_energy_terms,
                           float* h_gradients, int dstride, void* cuda_stream);

/* ADADELTA local search (R7) from each of n starting genotypes: d_genotypes device [n][gstride] in/out
 * (best genotype seen), d_energies device [n] out (its energy), d_iters device [n] out (evals used) or NULL,
 * d_trace device [n][params->lsit] out or NULL: the energy evaluated at iteration k (x_k before its step;
 * entries past the iterations performed are left untouched). */
int adock_local_search(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                       float* d_genotypes, int n, int gstride, float* d_energies, int* d_iters, float* d_trace,
                       void* cuda_stream);

/* adock_local_search for callers that may not allocate device memory (code under stream capture, serving loops,
 * harnesses that forbid cudaMalloc): the same ADADELTA search (R7), same arguments and outputs, on the
 * lane-per-individual kernel (8 warps per CTA, one chain per lane) whose per-chain state (best genotype, E[g^2],
 * E[dx^2]: 19 + 3R floats per chain) lives in a file-scope device array of ADOCK_NOALLOC_SCRATCH_BYTES inside the
 * library instead of a stream-ordered allocation.  Calls no cudaMalloc / cudaFree / allocating library routine; the
 * array's device address is looked up once per device (first call with that device current).
 * Limit: 32*ceil(n/32) chains, rounded up to whole CTAs, times (19 + 3R)*4 bytes must fit the array (R = 8: about
 * 97,000 chains; R = 64: about 19,000); a larger batch returns ADOCK_ELIMIT with the sizes in adock_last_error() and
 * launches nothing.  ADOCK_ELIMIT also if the ligand does not fit that kernel's shared memory.
 * Every GPU that loads the library holds the array until exit.  Every call shares it and finds the last call's
 * contents (the kernel initialises all state it reads: nothing needs clearing); calls that OVERLAP on the GPU
 * (different streams, or two host threads) race on it: serialise them.  Asynchronous on cuda_stream. */
#define ADOCK_NOALLOC_SCRATCH_BYTES (16u << 20)
int adock_local_search_noalloc(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                               float* d_genotypes, int n, int gstride, float* d_energies, int* d_iters, float* d_trace,
                               void* cuda_stream);

/* Solis-Wets local search (R11; Solis & Wets 1981) from each of n genotypes:
 * d_genotypes device [n][gstride] in/out (the accepted genotype), d_energies device [n] IN/OUT: on entry the energy
 * of each starting genotype (carried, not re-evaluated), on return the accepted energy; d_evals device [n] out
 * (evaluations used: 1 or 2 per iteration) or NULL; d_trace device [n][params->lsit] out or NULL: the accepted
 * energy after iteration k.  Chain i draws its steps from Philox (R8) with counter (it*ceil(D/4)+d/4, 6, i,
 * generation) and key seed.  Runs params->lsit iterations at most, whatever params->ls_method says. */
int adock_solis_wets(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params,
                     float* d_genotypes, int n, int gstride, float* d_energies, int* d_evals, float* d_trace,
                     unsigned long long seed, unsigned int generation, void* cuda_stream);

/* Philox4x32-10 (R8): out[i] = philox(key, ctr[i]); key host uint32[2], d_ctr/d_out device uint32 [n][4]. */
int adock_philox(const unsigned int key[2], const unsigned int* d_ctr, int n, unsigned int* d_out, void* cuda_stream);

/* One GA generation of `nrun` runs without scoring (R9), for bit-exact decision checks.  d_pop device
 * [nrun][P][G] (G = 7+R), d_energies device [nrun][P]; writes d_newpop [nrun][P][G] (slot 0 = elite),
 * d_decisions device int [nrun][P][10] = a1,a2,A,b1,b2,B,do_xover,p1,p2,mutation mask; d_ls_picks device
 * int [nrun][P] (first n_ls entries valid), *n_ls host.  generation >= 1. gen 0 with d_pop NULL:
 * writes the initial population into d_newpop. */
int adock_ga_generation(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params, int nrun, int P,
                        int generation, unsigned long long seed, const float* d_pop, const float* d_energies,
                        float* d_newpop, int* d_decisions, int* d_ls_picks, int* n_ls, void* cuda_stream);

/* Full LGA docking (R9): nrun independent runs of population pop_size until each
 * has used max_evals evaluations (checked per generation) or params->max_gens generations.  Outputs host:
 * best_genotypes [nrun][7+R], best_energies [nrun], best_coords [nrun][N][3] or NULL, evals_used [nrun]
 * or NULL, gens_used [nrun] or NULL.  Synchronous. */
int adock_dock(const adock_grids* grids, const adock_ligand* ligand, const adock_params* params, int nrun, int pop_size,
               long long max_evals, unsigned long long seed, float* best_genotypes, float* best_energies,
               float* best_coords, long long* evals_used, int* gens_used, void* cuda_stream);

/* Multi-ligand batch (one resident grid set, many ligands): docks nlig ligands
 * concurrently, every kernel launch covering all ligands and runs.  seeds host [nlig].  Output arrays host,
 * ligand-major, with per-ligand genotype stride gstride >= max_l(7+R_l) and coordinate stride
 * cstride >= max_l(N_l): best_genotypes [nlig][nrun][gstride], best_energies [nlig][nrun], best_coords
 * [nlig][nrun][cstride][3] or NULL, evals_used [nlig][nrun] or NULL, gens_used [nlig][nrun] or NULL (generations each
 * run lasted: below max_gens when the eval budget or autostop ended it).  Synchronous.
 * A ligand's result does not depend on what else is in the batch (same kernel variant: bit-identical to adock_dock of that
 * ligand and seed).  Launches with more CTAs than SMs take the ligands in order of decreasing estimated cost.  Environment
 * switch for measurements only: ADOCK_LS_QUEUE=1 runs the local search with one work queue per team of warps instead
 * (dock_ls_lane_queue_kernel; same results, profiles/r02_lane_variants.md). */
int adock_dock_many(const adock_grids* grids, const adock_ligand* const* ligands, int nlig, const adock_params* params,
                    int nrun, int pop_size, long long max_evals, const unsigned long long* seeds, int gstride,
                    float* best_genotypes, float* best_energies, int cstride, float* best_coords, long long* evals_used,
                    int* gens_used, void* cuda_stream);

/* Screening pipeline (Fig. 1: host-side ligand setup overlapped with the docking of
 * the previous ligand; lines 100-106: one resident grid set for all ligands).  Docks nlig ligands against one grid
 * set in batches of `batch` ligands (one adock_dock_many-style launch sequence per batch on cuda_stream; batch = 0:
 * the library sizes each batch to fill one wave of its local-search kernel on this device).  While
 * batch b is docked, host_threads worker threads run the ligand preprocessing (R2) of batch b+1 and its images are
 * uploaded from pinned memory on an internal copy stream, so the device never waits for the host except before the
 * first batch.  Ligands are dealt into batches by atom count (similar sizes share a launch); outputs keep the
 * caller's order.  ligs: host array of descriptors whose arrays are host and laid out as for adock_load_ligand;
 * force-field tables (T, pair_coeffs, solpar, vol) are shared by all ligands.  seeds host [nlig].  Outputs host:
 * best_genotypes [nlig][nrun][gstride] (gstride >= max(7+R)), best_energies [nlig][nrun], evals_used [nlig][nrun] or
 * NULL.  stats may be NULL.  A ligand the library rejects fails the whole call with that error (its index is in
 * adock_last_error).  Synchronous. */
typedef struct adock_ligand_desc {
    int N; const float* xyz; const int* type; const float* charge;
    int nbonds; const int* bonds; int R; const int* rot_bonds; int root_atom;
} adock_ligand_desc;
typedef struct adock_screen_stats {
    double wall_s;        /* whole call */
    double dock_s;        /* sum over batches of the time inside the docking call of that batch */
    double prep_s;        /* sum over batches of the host preprocessing + upload time (worker wall clock) */
    double exposed_s;     /* time the docking loop waited for a batch that was not ready (first batch included) */
    int batches;
    int host_threads;
} adock_screen_stats;
int adock_screen(const adock_grids* grids, const adock_params* params, int T, const float* pair_coeffs, const float* solpar,
                 const float* vol, int nlig, const adock_ligand_desc* ligs, int nrun, int pop_size, long long max_evals,
                 const unsigned long long* seeds, int batch, int host_threads, int gstride, float* best_genotypes,
                 float* best_energies, long long* evals_used, adock_screen_stats* stats, void* cuda_stream);

/* Pose post-processing (S8(f) NEXT-4; "root mean squared (Euclidean) distance (RMSD) ... between
 * the final best pose from docking and the crystallographic pose"; R13).  coords: host [n][N][3] (e.g. best_coords of
 * adock_dock), same atom order everywhere, no superposition, no symmetry correction.
 *   rmsd_ref  host [n] out or NULL: RMSD of pose k against ref (host [N][3]; required if rmsd_ref != NULL)
 *   rmsd_pair host [n][n] out or NULL: RMSD between poses a and b (symmetric, zero diagonal)
 *   cluster   host [n] out or NULL (needs energies host [n] and tol > 0): poses visited in order of increasing
 *             energy (ties: lower index); a pose joins the first cluster, in creation order, whose seed (its
 *             lowest-energy member) is within tol Angstrom RMSD, else it seeds cluster number *nclusters++ [LIT].
 * The distances are computed on the device (one warp per pose pair), the clustering on the host from them. */
int adock_pose_rmsd(int n, int N, const float* coords, const float* ref, float* rmsd_ref, float* rmsd_pair,
                    const float* energies, float tol, int* cluster, int* nclusters, void* cuda_stream);

/* Timing of the dominant kernel (the ADADELTA kernel of adock_dock / adock_dock_many) for roofline
 * accounting: while enabled, every launch of it is bracketed by CUDA events on the launching stream.
 * adock_profile(1) enables and resets, adock_profile(0) disables.  adock_profile_read returns the summed
 * duration (ms), the number of launches timed and the evaluations they performed (calling thread). */
int adock_profile(int enable);
int adock_profile_read(double* ls_ms, long long* ls_launches, long long* ls_evals);

/* Measured peak of the roofline that bounds the path (plain FP32 arithmetic, "bound": "alu"):
 * times a kernel of independent fma.rn.f32x2 chains (16 warps on every SM) on cuda_stream and returns the achieved
 * TFLOP/s (FMA = 2 FLOP) and FMA lanes per clock and SM at the device's nominal maximum clock (128 = one FP32 FMA per
 * lane and clock).  Synchronous.  MEASURED_PEAKS.json carries HBM and tensor figures only; bench.py reports this one. */
int adock_alu_peak(double* tflops, double* fma_lanes_per_clk_sm, void* cuda_stream);

/* Measurement behind the TM variants of the lane kernels (atom positions in tensor memory, addressed
 * thread i <-> lane i of the warp's quarter with a warp-uniform column): one CTA of `warps` (1..12) warps per SM.
 * mode 0: write / read-back of every column of every warp's slice with tcgen05.st / tcgen05.ld (.x1, and .x4 + .x2 at
 * columns 6m, the position layout): *errors = mismatches (must be 0).  mode 1 / 3: dependent-load latency of tensor memory /
 * shared memory, cycles per load.  mode 2 / 4: 8 independent 64-bit loads per iteration from tensor memory / shared memory,
 * cycles per iteration and warp.  Synchronous.  profiles/r02_tmem_scratch.md holds the numbers of this pool's B200. */
int adock_tmem_probe(int warps, int mode, int iters, int* errors, double* cycles_per_iteration, void* cuda_stream);

/* Kernel launches issued by this library on the calling thread since the last reset (bench accounting). */
long long adock_launch_count(int reset);

const char* adock_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ADOCK_H */
