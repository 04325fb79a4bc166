// oracle/adock_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, fp64 CPU statement of what the hot path of AutoDock-GPU-style LGA docking computes
// (arxiv 2007.03678; AutoDock4 energy function + Lamarckian GA; line 64: ADADELTA
// local search, nrun independent runs; line 116: affinity / electrostatic / desolvation grid maps).
// The paper gives no formulas; every formula below follows the reading fixed in DESIGN.md
// ("Readings", R1..R10, taken from SURVEY.md section 8(c) C1..C10; R11 Solis-Wets local search, lines
// 58/64/136 + Solis & Wets 1981; R12 autostop, line 197).  Written in the order and
// notation of those readings, no blocking, no fusion, no reordering.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use
// this file.  It shares no code with paper_2007_03678_b200/csrc (the CUDA path) and neither
// includes the other.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): identity pose, rigid-motion invariants,
// trilinear node/affine exactness + scipy map_coordinates, two-atom closed forms, brute-force pair
// enumeration, Newton's third law, central finite differences, ADADELTA first-step closed form and
// convergence on quadratics, Philox statistical/bijectivity checks (+ cuRAND on the GPU box),
// GA invariants and eval accounting, Solis-Wets contraction/expansion schedules and first two steps in
// closed form, autostop limits (tests/test_oracle_solis_wets.py).  Parity unpinned: per-run LGA trajectories beyond the first
// generations (chaotic; compared in distribution only).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <queue>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

// Precision of the SCORE path (R3-R6: pose, trilinear, grid_atom, pair_energy, score).  fp64 is the oracle.  Compiled a
// second time with -DORC_REAL=float (oracle/liboracle_f32.so) the very same statements run in honest fp32 (SURVEY.md
// section 8(c): "also a compile-time fp32 mode to measure how far honest fp32 lands from fp64 -- sets expectations
// for the GPU tolerance").  That build is a measuring stick for tolerances only; it is never the reference of a parity
// test.  Interfaces stay double in both builds; search (R7-R12) always runs in fp64 around the score.
#ifndef ORC_REAL
#define ORC_REAL double
#endif
typedef ORC_REAL real;

namespace {

const double PI = 3.14159265358979323846;

struct OPar {               // mirrors workloads.DEFAULT_PARAMS by name (own layout; not the CUDA struct)
    double elec_scale, diel_A, diel_B, diel_k, diel_lambda;
    double w_desolv, ds_sigma, qasp, r_min, k_wall;
    double ad_rho, ad_eps;
    double lsrat, tourn_prob, xover_rate, mut_rate, dmov, dang;
    // R11 Solis-Wets: initial / smallest step scale, expansion / contraction factors, bias update coefficients
    double sw_rho0, sw_rho_lb, sw_expand, sw_contract, sw_bias_keep, sw_bias_gain, sw_bias_decay;
    double as_tol;          // R12 autostop: threshold on the std-dev of a run's best energy over as_window generations
    int lsit, max_gens;
    int ls_method;          // 0 = ADADELTA (R7), 1 = Solis-Wets (R11)
    int sw_max_succ, sw_max_fail;
    int autostop, as_window;
};

struct OLig {
    int N = 0, R = 0, T = 0, nb = 0, root = 0, nfrag = 0;
    std::vector<double> x0;            // [N][3]
    std::vector<int> type;
    std::vector<double> q;
    std::vector<int> bonds;            // [nb][2]
    std::vector<int> ta, tb;           // oriented rotatable bonds: a_k root side, b_k moves
    std::vector<uint8_t> moved;        // [R][N]
    std::vector<int> depth, tor_order, frag, dist;
    double c[3] = {0, 0, 0};           // pivot
    std::vector<int> pairs;            // [np][2], lexicographic
    std::vector<double> coef;          // [T][T][4]
    std::vector<double> solpar, vol;
};

struct OGrid {
    int M = 0, nx = 0, ny = 0, nz = 0;
    double h = 0, org[3] = {0, 0, 0};
    std::vector<float> maps;           // [M][nz][ny][nx]
};

// ------------------------------------------------------------------ R2: ligand preprocessing
// reachable set from `start` over all bonds except bond index `skip` given as (sa,sb) (or -1)
std::vector<uint8_t> reach(const OLig& L, int start, int sa, int sb) {
    std::vector<uint8_t> seen(L.N, 0);
    std::queue<int> Q;
    seen[start] = 1;
    Q.push(start);
    while (!Q.empty()) {
        int u = Q.front();
        Q.pop();
        for (int b = 0; b < L.nb; ++b) {
            int p = L.bonds[2 * b], r = L.bonds[2 * b + 1];
            if ((p == sa && r == sb) || (p == sb && r == sa)) continue;
            int v = (p == u) ? r : (r == u) ? p : -1;
            if (v >= 0 && !seen[v]) { seen[v] = 1; Q.push(v); }
        }
    }
    return seen;
}

int prep(OLig& L, const int* rot) {
    const int N = L.N, R = L.R;
    // step 1: rigid fragments = components after deleting rotatable bonds; id = order of first atom
    auto is_rot = [&](int p, int r) {
        for (int k = 0; k < R; ++k)
            if ((rot[2 * k] == p && rot[2 * k + 1] == r) || (rot[2 * k] == r && rot[2 * k + 1] == p)) return true;
        return false;
    };
    L.frag.assign(N, -1);
    L.nfrag = 0;
    for (int s = 0; s < N; ++s) {
        if (L.frag[s] >= 0) continue;
        std::queue<int> Q;
        L.frag[s] = L.nfrag;
        Q.push(s);
        while (!Q.empty()) {
            int u = Q.front();
            Q.pop();
            for (int b = 0; b < L.nb; ++b) {
                int p = L.bonds[2 * b], r = L.bonds[2 * b + 1];
                if (is_rot(p, r)) continue;
                int v = (p == u) ? r : (r == u) ? p : -1;
                if (v >= 0 && L.frag[v] < 0) { L.frag[v] = L.nfrag; Q.push(v); }
            }
        }
        ++L.nfrag;
    }
    // steps 2,3: orient (a_k root side), moved set M_k
    L.ta.resize(R); L.tb.resize(R); L.moved.assign((size_t)R * N, 0);
    for (int k = 0; k < R; ++k) {
        int a = rot[2 * k], b = rot[2 * k + 1];
        bool bonded = false;
        for (int e = 0; e < L.nb; ++e)
            if ((L.bonds[2 * e] == a && L.bonds[2 * e + 1] == b) || (L.bonds[2 * e] == b && L.bonds[2 * e + 1] == a)) bonded = true;
        if (!bonded) return -1;
        std::vector<uint8_t> fromroot = reach(L, L.root, a, b);
        if (fromroot[a] && fromroot[b]) return -1;              // bond in a ring: not rotatable
        if (!fromroot[a]) std::swap(a, b);
        L.ta[k] = a; L.tb[k] = b;
        std::vector<uint8_t> m = reach(L, b, a, b);
        for (int i = 0; i < N; ++i) L.moved[(size_t)k * N + i] = m[i];
    }
    // step 3b: depth(k) = number of rotatable bonds on the path root -> b_k (k itself counts)
    L.depth.assign(R, 0);
    for (int k = 0; k < R; ++k)
        for (int k2 = 0; k2 < R; ++k2)
            if (L.moved[(size_t)k2 * N + L.tb[k]]) ++L.depth[k];
    // step 4: deepest first, ties by k ascending
    L.tor_order.resize(R);
    for (int k = 0; k < R; ++k) L.tor_order[k] = k;
    std::stable_sort(L.tor_order.begin(), L.tor_order.end(),
                     [&](int p, int r) { return L.depth[p] > L.depth[r]; });
    // step 5: pivot = fp64 mean rounded once to fp32
    for (int d = 0; d < 3; ++d) {
        double s = 0;
        for (int i = 0; i < N; ++i) s += L.x0[3 * i + d];
        L.c[d] = (double)(float)(s / N);
    }
    // step 6: topological distances by BFS
    L.dist.assign((size_t)N * N, 1 << 20);
    for (int s = 0; s < N; ++s) {
        std::queue<int> Q;
        L.dist[(size_t)s * N + s] = 0;
        Q.push(s);
        while (!Q.empty()) {
            int u = Q.front();
            Q.pop();
            for (int b = 0; b < L.nb; ++b) {
                int p = L.bonds[2 * b], r = L.bonds[2 * b + 1];
                int v = (p == u) ? r : (r == u) ? p : -1;
                if (v >= 0 && L.dist[(size_t)s * N + v] > L.dist[(size_t)s * N + u] + 1) {
                    L.dist[(size_t)s * N + v] = L.dist[(size_t)s * N + u] + 1;
                    Q.push(v);
                }
            }
        }
    }
    // step 7: pair (i<j) excluded iff d(i,j) <= 3 or rigid (no torsion separating i and j that has
    // neither i nor j on its axis)
    L.pairs.clear();
    for (int i = 0; i < N; ++i)
        for (int j = i + 1; j < N; ++j) {
            if (L.dist[(size_t)i * N + j] <= 3) continue;
            bool flexible = false;
            for (int k = 0; k < R; ++k) {
                bool sep = L.moved[(size_t)k * N + i] != L.moved[(size_t)k * N + j];
                bool on_axis = (i == L.ta[k] || i == L.tb[k] || j == L.ta[k] || j == L.tb[k]);
                if (sep && !on_axis) flexible = true;
            }
            if (flexible) { L.pairs.push_back(i); L.pairs.push_back(j); }
        }
    return 0;
}

// ------------------------------------------------------------------ small vector helpers
template <class F> inline void cross(const F* a, const F* b, F* o) {
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}
template <class F> inline F dot(const F* a, const F* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// Hamilton product p (x) q, components (w,x,y,z)
inline void qmul(const double* p, const double* q, double* o) {
    o[0] = p[0] * q[0] - p[1] * q[1] - p[2] * q[2] - p[3] * q[3];
    o[1] = p[0] * q[1] + p[1] * q[0] + p[2] * q[3] - p[3] * q[2];
    o[2] = p[0] * q[2] - p[1] * q[3] + p[2] * q[0] + p[3] * q[1];
    o[3] = p[0] * q[3] + p[1] * q[2] - p[2] * q[1] + p[3] * q[0];
}

inline double wrap_pi(double a) { return a - 2 * PI * std::floor((a + PI) / (2 * PI)); }

// ------------------------------------------------------------------ R3: pose builder
// g = (t[3], q[4] = w,x,y,z, tau[R]).  Returns false for |q| < 1e-12.
bool pose(const OLig& L, const double* g, real* x) {
    const int N = L.N;
    std::vector<real> y(L.x0.begin(), L.x0.end());
    for (int o = 0; o < L.R; ++o) {                       // deepest first: reference-frame axes valid
        int k = L.tor_order[o];
        const real xa[3] = {(real)L.x0[3 * L.ta[k]], (real)L.x0[3 * L.ta[k] + 1], (real)L.x0[3 * L.ta[k] + 2]};
        const real xb[3] = {(real)L.x0[3 * L.tb[k]], (real)L.x0[3 * L.tb[k] + 1], (real)L.x0[3 * L.tb[k] + 2]};
        real u[3] = {xb[0] - xa[0], xb[1] - xa[1], xb[2] - xa[2]};
        real n = std::sqrt(dot(u, u));
        for (real& c : u) c /= n;
        real ct = std::cos((real)g[7 + k]), st = std::sin((real)g[7 + k]);
        for (int i = 0; i < N; ++i) {
            if (!L.moved[(size_t)k * N + i]) continue;
            real v[3] = {y[3 * i] - xa[0], y[3 * i + 1] - xa[1], y[3 * i + 2] - xa[2]};
            real uxv[3];
            cross(u, v, uxv);
            real ud = dot(u, v);
            for (int d = 0; d < 3; ++d)                   // Rodrigues, right-hand about a->b
                y[3 * i + d] = xa[d] + v[d] * ct + uxv[d] * st + u[d] * ud * (1 - ct);
        }
    }
    const real q0 = (real)g[3], q1 = (real)g[4], q2 = (real)g[5], q3 = (real)g[6];
    real qn = std::sqrt(q0 * q0 + q1 * q1 + q2 * q2 + q3 * q3);
    if (!(qn >= (real)1e-12)) return false;
    real w = q0 / qn, a = q1 / qn, b = q2 / qn, c = q3 / qn;
    real Rm[9] = {1 - 2 * (b * b + c * c), 2 * (a * b - w * c),     2 * (a * c + w * b),
                  2 * (a * b + w * c),     1 - 2 * (a * a + c * c), 2 * (b * c - w * a),
                  2 * (a * c - w * b),     2 * (b * c + w * a),     1 - 2 * (a * a + b * b)};
    for (int i = 0; i < N; ++i) {
        real v[3] = {y[3 * i] - (real)L.c[0], y[3 * i + 1] - (real)L.c[1], y[3 * i + 2] - (real)L.c[2]};
        for (int d = 0; d < 3; ++d) x[3 * i + d] = (real)g[d] + Rm[3 * d] * v[0] + Rm[3 * d + 1] * v[1] + Rm[3 * d + 2] * v[2];
    }
    return true;
}

// ------------------------------------------------------------------ R4: grid term
// trilinear value and gradient (per Angstrom) of map m at point p, clamp + floor rule.
// margin (optional) = min over in-box axes of the distance (grid units) to the nearest cell face.
real trilinear(const OGrid& G, int m, const real* p, real* grad, real* outside /*[3] u-uc*/, double* margin) {
    const int n[3] = {G.nx, G.ny, G.nz};
    int i0[3];
    real f[3];
    for (int d = 0; d < 3; ++d) {
        real u = (p[d] - (real)G.org[d]) / (real)G.h;
        real uc = std::min(std::max(u, (real)0.0), (real)(n[d] - 1));
        i0[d] = std::min((int)std::floor(uc), n[d] - 2);
        f[d] = uc - i0[d];
        if (outside) outside[d] = u - uc;
        if (margin)      // gradient kinks sit at integer u (cell faces, box faces)
            *margin = std::min(*margin, (double)((u != uc) ? std::fabs(u - uc) : std::fabs(u - std::round(u))));
    }
    const float* map = &G.maps[(size_t)m * G.nz * G.ny * G.nx];
    real val = 0, gx = 0, gy = 0, gz = 0;
    for (int cz = 0; cz < 2; ++cz)
        for (int cy = 0; cy < 2; ++cy)
            for (int cx = 0; cx < 2; ++cx) {
                real v = map[((size_t)(i0[2] + cz) * G.ny + (i0[1] + cy)) * G.nx + (i0[0] + cx)];
                real wx = cx ? f[0] : 1 - f[0], wy = cy ? f[1] : 1 - f[1], wz = cz ? f[2] : 1 - f[2];
                val += wz * wy * wx * v;
                gx += wz * wy * (cx ? (real)1.0 : (real)-1.0) * v;
                gy += wz * (cy ? (real)1.0 : (real)-1.0) * wx * v;
                gz += (cz ? (real)1.0 : (real)-1.0) * wy * wx * v;
            }
    if (grad) { grad[0] = gx / (real)G.h; grad[1] = gy / (real)G.h; grad[2] = gz / (real)G.h; }
    return val;
}

// E_i and g_i of atom i at x (R4): type map + q*elec + |q|*desolv + linear wall outside the box
real grid_atom(const OGrid& G, const OPar& P, int type, real q, int T, const real* x, real* g, double* margin) {
    real gt[3], ge[3], gd[3], out[3];
    real vt = trilinear(G, type, x, gt, out, margin);
    real ve = trilinear(G, T, x, ge, nullptr, nullptr);
    real vd = trilinear(G, T + 1, x, gd, nullptr, nullptr);
    real E = vt + q * ve + std::fabs(q) * vd;
    for (int d = 0; d < 3; ++d) {
        if (out[d] != 0.0) {                    // violated axis: interpolant constant along it
            E += (real)P.k_wall * (real)G.h * std::fabs(out[d]);
            g[d] = (real)P.k_wall * (out[d] > 0 ? (real)1.0 : (real)-1.0);
        } else {
            g[d] = gt[d] + q * ge[d] + std::fabs(q) * gd[d];
        }
    }
    return E;
}

// ------------------------------------------------------------------ R5: intramolecular pair term
// energy and dE/dr of one pair at separation d (before the r_min floor); dsco = S_i V_j + S_j V_i
real pair_energy(const OPar& P, real c12, real cA, real expA, real qq, real dsco, real d, real* dEdr) {
    const real r_min = (real)P.r_min, A = (real)P.diel_A, B = (real)P.diel_B, k = (real)P.diel_k, lam = (real)P.diel_lambda;
    const real sig = (real)P.ds_sigma;
    real r = std::max(d, r_min);
    real e_vdw = c12 / std::pow(r, (real)12) - cA / std::pow(r, expA);
    real d_vdw = -12 * c12 / std::pow(r, (real)13) + expA * cA / std::pow(r, expA + 1);
    real ex = std::exp(-lam * B * r);
    real eps = A + B / (1 + k * ex);
    real deps = B * k * lam * B * ex / ((1 + k * ex) * (1 + k * ex));
    real e_el = (real)P.elec_scale * qq / (eps * r);
    real d_el = -(real)P.elec_scale * qq * (deps * r + eps) / ((eps * r) * (eps * r));
    real e_ds = (real)P.w_desolv * dsco * std::exp(-r * r / (2 * sig * sig));
    real d_ds = -(r / (sig * sig)) * e_ds;
    if (dEdr) *dEdr = (d < r_min) ? (real)0.0 : d_vdw + d_el + d_ds;
    return e_vdw + e_el + e_ds;
}

// ------------------------------------------------------------------ R4-R6: full score of one genotype
// grad (may be null): [dE/dt (3), dE/domega (3), dE/dtau (R)]; terms: [inter, intra];
// margins (may be null): [min face distance in grid units, min | |x_i-x_j| - r_min | in Angstrom]
// scales (may be null): [S_t, S_omega, S_tau] = sums of the MAGNITUDES of the terms that are added up in
// each gradient block (conditioning of the sums; used only to set test tolerances, R10)
double score(const OGrid& G, const OLig& L, const OPar& P, const double* g, double* grad, double* terms, double* margins,
             double* scales = nullptr) {
    const int N = L.N;
    const double nan = std::numeric_limits<double>::quiet_NaN();
    std::vector<real> x(3 * N), f(3 * N, (real)0.0), fabs_i(N, (real)0.0);
    if (!pose(L, g, x.data())) {
        if (grad) for (int d = 0; d < 6 + L.R; ++d) grad[d] = nan;
        if (terms) terms[0] = terms[1] = nan;
        return nan;
    }
    const real gt[3] = {(real)g[0], (real)g[1], (real)g[2]};
    double fm = 1.0, pm = 1e30;
    real e_inter = 0, e_intra = 0;
    for (int i = 0; i < N; ++i) {
        e_inter += grid_atom(G, P, L.type[i], (real)L.q[i], L.T, &x[3 * i], &f[3 * i], &fm);
        fabs_i[i] = std::sqrt(dot(&f[3 * i], &f[3 * i]));
    }
    const size_t np = L.pairs.size() / 2;
    for (size_t p = 0; p < np; ++p) {
        int i = L.pairs[2 * p], j = L.pairs[2 * p + 1];
        int ti = L.type[i], tj = L.type[j];
        const double* co = &L.coef[((size_t)ti * L.T + tj) * 4];
        real Si = (real)L.solpar[ti] + (real)P.qasp * std::fabs((real)L.q[i]), Sj = (real)L.solpar[tj] + (real)P.qasp * std::fabs((real)L.q[j]);
        real dsco = Si * (real)L.vol[tj] + Sj * (real)L.vol[ti];
        real dv[3] = {x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2]};
        real d = std::sqrt(dot(dv, dv)), dEdr;
        e_intra += pair_energy(P, (real)co[0], (real)co[1], (real)co[2], (real)L.q[i] * (real)L.q[j], dsco, d, &dEdr);
        pm = std::min(pm, (double)std::fabs(d - (real)P.r_min));
        if (d >= (real)P.r_min) {
            for (int c = 0; c < 3; ++c) {
                f[3 * i + c] += dEdr * dv[c] / d;
                f[3 * j + c] -= dEdr * dv[c] / d;
            }
            fabs_i[i] += std::fabs(dEdr);
            fabs_i[j] += std::fabs(dEdr);
        }
    }
    if (scales) {
        scales[0] = scales[1] = scales[2] = 0;
        for (int i = 0; i < N; ++i) {
            real rel[3] = {x[3 * i] - gt[0], x[3 * i + 1] - gt[1], x[3 * i + 2] - gt[2]};
            scales[0] += fabs_i[i];
            scales[1] += std::sqrt(dot(rel, rel)) * fabs_i[i];
        }
        for (int k = 0; k < L.R; ++k) {
            double sk = 0;
            for (int i = 0; i < N; ++i) {
                if (!L.moved[(size_t)k * N + i]) continue;
                real rel[3] = {x[3 * i] - x[3 * L.ta[k]], x[3 * i + 1] - x[3 * L.ta[k] + 1], x[3 * i + 2] - x[3 * L.ta[k] + 2]};
                sk += std::sqrt(dot(rel, rel)) * fabs_i[i];
            }
            scales[2] += sk * sk;
        }
        scales[2] = std::sqrt(scales[2]);
    }
    if (terms) { terms[0] = e_inter; terms[1] = e_intra; }
    if (margins) { margins[0] = fm; margins[1] = pm; }
    if (grad) {                                            // R6: back-propagation
        std::vector<real> gr(6 + L.R, (real)0.0);
        for (int i = 0; i < N; ++i) {
            real rel[3] = {x[3 * i] - gt[0], x[3 * i + 1] - gt[1], x[3 * i + 2] - gt[2]}, t[3];
            cross(rel, &f[3 * i], t);
            for (int d = 0; d < 3; ++d) { gr[d] += f[3 * i + d]; gr[3 + d] += t[d]; }
        }
        for (int k = 0; k < L.R; ++k) {
            const real* xa = &x[3 * L.ta[k]];
            const real* xb = &x[3 * L.tb[k]];
            real u[3] = {xb[0] - xa[0], xb[1] - xa[1], xb[2] - xa[2]};
            real n = std::sqrt(dot(u, u));
            for (real& c : u) c /= n;
            real tq[3] = {0, 0, 0};
            for (int i = 0; i < N; ++i) {
                if (!L.moved[(size_t)k * N + i]) continue;
                real rel[3] = {x[3 * i] - xa[0], x[3 * i + 1] - xa[1], x[3 * i + 2] - xa[2]}, t[3];
                cross(rel, &f[3 * i], t);
                for (int d = 0; d < 3; ++d) tq[d] += t[d];
            }
            gr[6 + k] = dot(u, tq);
        }
        for (int d = 0; d < 6 + L.R; ++d) grad[d] = gr[d];
    }
    return e_inter + e_intra;
}

// ------------------------------------------------------------------ R7: ADADELTA (Zeiler), generic update
// one update from gradient gr[D]: accumulators Eg2, Ed2 in place, step written to delta
void adadelta_update(int D, const double* gr, double* Eg2, double* Ed2, double rho, double eps, double* delta) {
    for (int d = 0; d < D; ++d) {
        Eg2[d] = rho * Eg2[d] + (1 - rho) * gr[d] * gr[d];
        delta[d] = -std::sqrt(Ed2[d] + eps) / std::sqrt(Eg2[d] + eps) * gr[d];
        Ed2[d] = rho * Ed2[d] + (1 - rho) * delta[d] * delta[d];
    }
}

// apply a step delta = (dt, domega, dtau) to genotype x (R7 last line)
void apply_step(int R, double* x, const double* delta) {
    for (int d = 0; d < 3; ++d) x[d] += delta[d];
    const double* w = delta + 3;
    double th = std::sqrt(dot(w, w));
    double dq[4] = {std::cos(th / 2), 0, 0, 0};
    double s = (th > 1e-12) ? std::sin(th / 2) / th : 0.5;
    for (int d = 0; d < 3; ++d) dq[1 + d] = s * w[d];
    double qn = std::sqrt(x[3] * x[3] + x[4] * x[4] + x[5] * x[5] + x[6] * x[6]);
    double qh[4] = {x[3] / qn, x[4] / qn, x[5] / qn, x[6] / qn}, o[4];
    qmul(dq, qh, o);
    double on = std::sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2] + o[3] * o[3]);
    for (int d = 0; d < 4; ++d) x[3 + d] = o[d] / on;
    for (int k = 0; k < R; ++k) x[7 + k] = wrap_pi(x[7 + k] + delta[6 + k]);
}

// docking local search: returns iterations (= evals) used; x and E updated to the best seen
int adadelta_dock(const OGrid& G, const OLig& L, const OPar& P, double* x, double* E, double* traceE, double* traceX) {
    const int R = L.R, D = 6 + R, Gn = 7 + R;
    std::vector<double> cur(x, x + Gn), best(x, x + Gn), Eg2(D, 0.0), Ed2(D, 0.0), gr(D), delta(D);
    double bestE = std::numeric_limits<double>::infinity();
    int it = 0;
    while (it < P.lsit) {
        double e = score(G, L, P, cur.data(), gr.data(), nullptr, nullptr);
        if (traceE) traceE[it] = e;
        if (traceX) std::copy(cur.begin(), cur.end(), traceX + (size_t)it * Gn);
        ++it;
        bool ok = std::isfinite(e);
        for (int d = 0; d < D; ++d) ok = ok && std::isfinite(gr[d]);
        if (!ok) break;
        if (e < bestE) { bestE = e; best = cur; }
        adadelta_update(D, gr.data(), Eg2.data(), Ed2.data(), P.ad_rho, P.ad_eps, delta.data());
        apply_step(R, cur.data(), delta.data());
    }
    if (std::isfinite(bestE)) { std::copy(best.begin(), best.end(), x); *E = bestE; }
    return it;
}

// ------------------------------------------------------------------ R8: Philox4x32-10 (Salmon et al. 2011)
inline void philox(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { P_INIT = 0, P_TOURN_A = 1, P_TOURN_B = 2, P_XOVER = 3, P_MUT = 4, P_LS_PICK = 5 };

// counter = (draw_index, purpose, individual id, generation); key = (seed lo, seed hi)
inline void draw4(uint64_t seed, uint32_t draw, uint32_t purpose, uint32_t id, uint32_t gen, uint32_t out[4]) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, ctr[4] = {draw, purpose, id, gen};
    philox(key, ctr, out);
}
inline double u01(uint32_t x) { return (double)(x >> 8) * (1.0 / 16777216.0); }          // exact, in [0,1)
inline int below(uint32_t x, int n) { return (int)std::floor(u01(x) * n); }               // floor(u*n), exact in fp64

// ------------------------------------------------------------------ R11: Solis-Wets local search
// PAPER.md lines 58, 64, 136 name the method and cite Solis & Wets 1981 [27] ("Minimization by random search
// techniques", the variant with an adaptive step scale and a bias vector); constants [LIT] -> params.  One iteration:
//   delta_d = rho * amp_d * (2 u_d - 1) + b_d        u_d: Philox word d&3 of draw (it*ceil(D/4) + d/4, P_SW, id, gen)
//   E(x (+) delta) < E : accept, b <- keep b + gain delta, success
//   else E(x (-) delta) < E : accept, b <- keep b - gain delta, success          (second evaluation only in this branch)
//   else b <- decay b, failure
//   sw_max_succ successes in a row: rho *= expand ; sw_max_fail failures in a row: rho *= contract
// until it == lsit or rho < rho_lb.  (+) is the step application of R7 (translation, left rotation by the rotation
// vector, wrapped torsions); amp = dmov for the translation, dang for the rotation vector and the torsions.
// E(x) is the carried energy (no evaluation).  A non-finite trial energy is a failure (comparison false).
struct SwFn { virtual double operator()(const double* x) = 0; virtual void step(double* x, const double* delta, double sign) = 0; virtual ~SwFn() {} };
enum { P_SW = 6 };
// returns evaluations used; x, E updated in place; iters = iterations done; rho_out = final step scale
int solis_wets(SwFn& f, int n, int D, const double* amp, const OPar& P, uint64_t seed, uint32_t id, uint32_t gen, double* x, double* E,
               int* iters, double* rho_out, double* traceE) {
    std::vector<double> b(D, 0.0), delta(D), cand(n);
    double rho = P.sw_rho0;
    int ns = 0, nf = 0, it = 0, evals = 0;
    const int nq = (D + 3) / 4;
    while (it < P.lsit && !(rho < P.sw_rho_lb)) {
        for (int q = 0; q < nq; ++q) {
            uint32_t r[4];
            draw4(seed, (uint32_t)(it * nq + q), P_SW, id, gen, r);
            for (int w = 0; w < 4 && 4 * q + w < D; ++w) delta[4 * q + w] = rho * amp[4 * q + w] * (2.0 * u01(r[w]) - 1.0) + b[4 * q + w];
        }
        std::copy(x, x + n, cand.begin());
        f.step(cand.data(), delta.data(), +1.0);
        double e = f(cand.data());
        ++evals;
        bool ok = false;
        if (e < *E) {
            for (int d = 0; d < D; ++d) b[d] = P.sw_bias_keep * b[d] + P.sw_bias_gain * delta[d];
            ok = true;
        } else {
            std::copy(x, x + n, cand.begin());
            f.step(cand.data(), delta.data(), -1.0);
            e = f(cand.data());
            ++evals;
            if (e < *E) {
                for (int d = 0; d < D; ++d) b[d] = P.sw_bias_keep * b[d] - P.sw_bias_gain * delta[d];
                ok = true;
            } else {
                for (int d = 0; d < D; ++d) b[d] = P.sw_bias_decay * b[d];
            }
        }
        if (ok) { std::copy(cand.begin(), cand.end(), x); *E = e; ++ns; nf = 0; } else { ++nf; ns = 0; }
        if (ns >= P.sw_max_succ) { rho *= P.sw_expand; ns = 0; }
        else if (nf >= P.sw_max_fail) { rho *= P.sw_contract; nf = 0; }
        if (traceE) traceE[it] = *E;
        ++it;
    }
    if (iters) *iters = it;
    if (rho_out) *rho_out = rho;
    return evals;
}

// ------------------------------------------------------------------ R9: GA
void ga_init_one(const OGrid& G, int R, uint64_t seed, uint32_t id, double* g) {
    uint32_t r[4];
    const int n[3] = {G.nx, G.ny, G.nz};
    draw4(seed, 0, P_INIT, id, 0, r);
    for (int d = 0; d < 3; ++d) g[d] = G.org[d] + u01(r[d]) * (G.h * (n[d] - 1));
    draw4(seed, 1, P_INIT, id, 0, r);                       // Shoemake uniform rotation
    double u1 = u01(r[0]), u2 = u01(r[1]), u3 = u01(r[2]);
    double s1 = std::sqrt(1 - u1), s2 = std::sqrt(u1);
    g[3] = s2 * std::cos(2 * PI * u3);
    g[4] = s1 * std::sin(2 * PI * u2);
    g[5] = s1 * std::cos(2 * PI * u2);
    g[6] = s2 * std::sin(2 * PI * u3);
    for (int k = 0; k < R; ++k) {
        if (k % 4 == 0) draw4(seed, 2 + k / 4, P_INIT, id, 0, r);
        g[7 + k] = -PI + 2 * PI * u01(r[k % 4]);
    }
}

// binary tournament: two uniform slots; with prob tourn_prob keep the lower-energy one else the other
int tournament(const OPar& P, int Pn, const double* E, uint64_t seed, uint32_t purpose, uint32_t id, uint32_t gen, int* dec) {
    uint32_t r[4];
    draw4(seed, 0, purpose, id, gen, r);
    int s1 = below(r[0], Pn), s2 = below(r[1], Pn);
    int lo = (E[s1] <= E[s2]) ? s1 : s2, hi = (E[s1] <= E[s2]) ? s2 : s1;
    int pick = (u01(r[2]) < P.tourn_prob) ? lo : hi;
    dec[0] = s1; dec[1] = s2; dec[2] = pick;
    return pick;
}

// next generation of one run.  dec: [P][10] = a1,a2,A, b1,b2,B, do_xover, p1, p2, mutation bitmask(low 31 blocks)
// newE[0] = carried elite energy; newE[s>0] = NaN (to be scored by the caller).
void ga_offspring(const OPar& P, int Pn, int R, int run, int gen, uint64_t seed, const double* pop, const double* E,
                  double* newpop, double* newE, int* dec) {
    const int Gn = 7 + R, NB = 4 + R;                       // gene blocks: tx,ty,tz,q,tau_1..tau_R
    int elite = 0;
    for (int s = 1; s < Pn; ++s) if (E[s] < E[elite]) elite = s;      // ties -> lowest slot
    std::copy(pop + (size_t)elite * Gn, pop + (size_t)(elite + 1) * Gn, newpop);
    newE[0] = E[elite];
    if (dec) { std::fill(dec, dec + 10, 0); dec[2] = elite; }
    for (int s = 1; s < Pn; ++s) {
        uint32_t id = (uint32_t)(run * Pn + s), r[4];
        int d[10] = {0};
        int A = tournament(P, Pn, E, seed, P_TOURN_A, id, gen, d);
        int B = tournament(P, Pn, E, seed, P_TOURN_B, id, gen, d + 3);
        double* c = newpop + (size_t)s * Gn;
        std::copy(pop + (size_t)A * Gn, pop + (size_t)(A + 1) * Gn, c);
        draw4(seed, 0, P_XOVER, id, gen, r);
        int c1 = below(r[1], NB + 1), c2 = below(r[2], NB + 1);
        int p1 = std::min(c1, c2), p2 = std::max(c1, c2);
        bool xo = u01(r[0]) < P.xover_rate;
        d[6] = xo; d[7] = p1; d[8] = p2;
        auto blk = [&](int b, int& lo, int& hi) {            // gene range of block b
            if (b < 3) { lo = b; hi = b + 1; } else if (b == 3) { lo = 3; hi = 7; } else { lo = 4 + b - 1; hi = lo + 1; }
        };
        if (xo)
            for (int b = p1; b < p2; ++b) {
                int lo, hi;
                blk(b, lo, hi);
                for (int gI = lo; gI < hi; ++gI) c[gI] = pop[(size_t)B * Gn + gI];
            }
        for (int b = 0; b < NB; ++b) {
            draw4(seed, b, P_MUT, id, gen, r);
            if (!(u01(r[0]) < P.mut_rate)) continue;
            if (b < 31) d[9] |= 1 << b;
            double amt = 2 * u01(r[1]) - 1;
            if (b < 3) {
                c[b] += amt * P.dmov;
            } else if (b == 3) {
                double ang = amt * P.dang, z = 2 * u01(r[2]) - 1, ph = 2 * PI * u01(r[3]);
                double sxy = std::sqrt(std::max(0.0, 1 - z * z));
                double dq[4] = {std::cos(ang / 2), std::sin(ang / 2) * sxy * std::cos(ph), std::sin(ang / 2) * sxy * std::sin(ph), std::sin(ang / 2) * z};
                double qn = std::sqrt(c[3] * c[3] + c[4] * c[4] + c[5] * c[5] + c[6] * c[6]);
                double qh[4] = {c[3] / qn, c[4] / qn, c[5] / qn, c[6] / qn}, o[4];
                qmul(dq, qh, o);
                double on = std::sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2] + o[3] * o[3]);
                for (int q4 = 0; q4 < 4; ++q4) c[3 + q4] = o[q4] / on;
            } else {
                c[4 + b - 1] = wrap_pi(c[4 + b - 1] + amt * P.dang);
            }
        }
        newE[s] = std::numeric_limits<double>::quiet_NaN();
        if (dec) std::copy(d, d + 10, dec + (size_t)s * 10);
    }
}

// local-search subset of one run in one generation: slot 0 + first n_ls-1 of a partial Fisher-Yates of 1..P-1
int ls_pick(const OPar& P, int Pn, int run, int gen, uint64_t seed, int* picks) {
    int n_ls = std::min(Pn, (int)std::ceil(P.lsrat * Pn - 1e-9));
    if (n_ls <= 0) return 0;
    std::vector<int> arr(Pn - 1);
    for (int s = 1; s < Pn; ++s) arr[s - 1] = s;
    picks[0] = 0;
    uint32_t r[4];
    for (int m = 0; m < n_ls - 1; ++m) {
        if (m % 4 == 0) draw4(seed, m / 4, P_LS_PICK, (uint32_t)(run * Pn), gen, r);
        int j = m + below(r[m % 4], Pn - 1 - m);
        std::swap(arr[m], arr[j]);
        picks[1 + m] = arr[m];
    }
    return n_ls;
}

struct SwDock : SwFn {
    const OGrid& G; const OLig& L; const OPar& P;
    SwDock(const OGrid& g, const OLig& l, const OPar& p) : G(g), L(l), P(p) {}
    double operator()(const double* x) override { return score(G, L, P, x, nullptr, nullptr, nullptr); }
    void step(double* x, const double* delta, double sign) override {
        std::vector<double> d(delta, delta + 6 + L.R);
        for (auto& v : d) v *= sign;
        apply_step(L.R, x, d.data());
    }
};
int solis_wets_dock(const OGrid& G, const OLig& L, const OPar& P, uint64_t seed, uint32_t id, uint32_t gen, double* x, double* E,
                    int* iters, double* rho_out, double* traceE) {
    const int D = 6 + L.R;
    std::vector<double> amp(D, P.dang);
    amp[0] = amp[1] = amp[2] = P.dmov;
    SwDock f(G, L, P);
    return solis_wets(f, 7 + L.R, D, amp.data(), P, seed, id, gen, x, E, iters, rho_out, traceE);
}

// R12 autostop ("stop ... if no progress is being made"; criterion [CHOICE] -> params): a run ends
// after generation g >= as_window when the population std-dev of its best energy over the last as_window generations
// is < as_tol.
bool autostop_hit(const OPar& P, const std::vector<double>& best_hist) {
    const int W = P.as_window;
    if (!P.autostop || W < 1 || (int)best_hist.size() < W) return false;
    double m = 0, v = 0;
    for (int i = 0; i < W; ++i) m += best_hist[best_hist.size() - W + i];
    m /= W;
    for (int i = 0; i < W; ++i) { const double d = best_hist[best_hist.size() - W + i] - m; v += d * d; }
    return std::sqrt(v / W) < P.as_tol;
}

struct RunResult { std::vector<double> best; double bestE; long long evals; int gens; };

RunResult dock_run(const OGrid& G, const OLig& L, const OPar& P, int run, int Pn, long long max_evals, uint64_t seed,
                   std::vector<double>* history) {
    const int R = L.R, Gn = 7 + R;
    std::vector<double> pop((size_t)Pn * Gn), E(Pn), npop((size_t)Pn * Gn), nE(Pn);
    std::vector<int> picks(Pn);
    for (int s = 0; s < Pn; ++s) {
        ga_init_one(G, R, seed, (uint32_t)(run * Pn + s), &pop[(size_t)s * Gn]);
        E[s] = score(G, L, P, &pop[(size_t)s * Gn], nullptr, nullptr, nullptr);
    }
    long long evals = Pn;
    int gen = 0;
    std::vector<double> best_hist;                          // per generation >= 1 (R12)
    if (history) history->push_back(*std::min_element(E.begin(), E.end()));
    while (evals < max_evals && gen < P.max_gens) {
        ++gen;
        ga_offspring(P, Pn, R, run, gen, seed, pop.data(), E.data(), npop.data(), nE.data(), nullptr);
        for (int s = 1; s < Pn; ++s) nE[s] = score(G, L, P, &npop[(size_t)s * Gn], nullptr, nullptr, nullptr);
        evals += Pn - 1;
        int n_ls = ls_pick(P, Pn, run, gen, seed, picks.data());
        for (int l = 0; l < n_ls; ++l) {                    // Lamarckian write-back
            double* xl = &npop[(size_t)picks[l] * Gn];
            if (P.ls_method == 1)
                evals += solis_wets_dock(G, L, P, seed, (uint32_t)(run * Pn + picks[l]), (uint32_t)gen, xl, &nE[picks[l]], nullptr, nullptr, nullptr);
            else
                evals += adadelta_dock(G, L, P, xl, &nE[picks[l]], nullptr, nullptr);
        }
        pop.swap(npop);
        E.swap(nE);
        best_hist.push_back(*std::min_element(E.begin(), E.end()));
        if (history) history->push_back(best_hist.back());
        if (autostop_hit(P, best_hist)) break;
    }
    int b = 0;
    for (int s = 1; s < Pn; ++s) if (E[s] < E[b]) b = s;
    RunResult r;
    r.best.assign(pop.begin() + (size_t)b * Gn, pop.begin() + (size_t)(b + 1) * Gn);
    r.bestE = E[b]; r.evals = evals; r.gens = gen;
    return r;
}

}  // namespace

// =================================================================== C interface for ctypes
extern "C" {

int orc_lig_create(int N, const float* xyz, const int* type, const float* charge, int nbonds, const int* bonds, int R,
                   const int* rot, int root, int T, const float* coeffs, const float* solpar, const float* vol, void** out) {
    if (N < 1 || R < 0 || T < 1 || root < 0 || root >= N) return -1;
    OLig* L = new OLig;
    L->N = N; L->R = R; L->T = T; L->nb = nbonds; L->root = root;
    L->x0.assign(xyz, xyz + 3 * N);
    L->type.assign(type, type + N);
    L->q.assign(charge, charge + N);
    L->bonds.assign(bonds, bonds + 2 * nbonds);
    L->coef.assign(coeffs, coeffs + (size_t)T * T * 4);
    L->solpar.assign(solpar, solpar + T);
    L->vol.assign(vol, vol + T);
    for (int i = 0; i < N; ++i) if (type[i] < 0 || type[i] >= T) { delete L; return -1; }
    for (int b = 0; b < 2 * nbonds; ++b) if (bonds[b] < 0 || bonds[b] >= N) { delete L; return -1; }
    if (prep(*L, rot) != 0) { delete L; return -1; }
    *out = L;
    return 0;
}
void orc_lig_free(void* p) { delete (OLig*)p; }

int orc_lig_info(void* p, int* npairs, int* nfrag) {
    OLig* L = (OLig*)p;
    *npairs = (int)(L->pairs.size() / 2);
    *nfrag = L->nfrag;
    return 0;
}
int orc_lig_get(void* p, int* pairs, int* tor_order, uint8_t* moved, int* depth, int* frag, int* rot_oriented, double* pivot, int* dist) {
    OLig* L = (OLig*)p;
    if (pairs) std::copy(L->pairs.begin(), L->pairs.end(), pairs);
    if (tor_order) std::copy(L->tor_order.begin(), L->tor_order.end(), tor_order);
    if (moved) std::copy(L->moved.begin(), L->moved.end(), moved);
    if (depth) std::copy(L->depth.begin(), L->depth.end(), depth);
    if (frag) std::copy(L->frag.begin(), L->frag.end(), frag);
    if (rot_oriented) for (int k = 0; k < L->R; ++k) { rot_oriented[2 * k] = L->ta[k]; rot_oriented[2 * k + 1] = L->tb[k]; }
    if (pivot) std::copy(L->c, L->c + 3, pivot);
    if (dist) std::copy(L->dist.begin(), L->dist.end(), dist);
    return 0;
}

int orc_grid_create(const float* maps, int M, int nx, int ny, int nz, double spacing, const float* origin, void** out) {
    if (M < 3 || nx < 2 || ny < 2 || nz < 2 || !(spacing > 0)) return -1;
    OGrid* G = new OGrid;
    G->M = M; G->nx = nx; G->ny = ny; G->nz = nz; G->h = spacing;
    for (int d = 0; d < 3; ++d) G->org[d] = origin[d];
    G->maps.assign(maps, maps + (size_t)M * nz * ny * nx);
    *out = G;
    return 0;
}
void orc_grid_free(void* p) { delete (OGrid*)p; }

int orc_pose(void* lig, const double* geno, double* xyz) {
    OLig* L = (OLig*)lig;
    std::vector<real> x(3 * L->N);
    if (!pose(*L, geno, x.data())) return -1;
    std::copy(x.begin(), x.end(), xyz);
    return 0;
}

int orc_trilinear(void* grid, int m, const double* xyz, int n, double* val, double* grad) {
    OGrid* G = (OGrid*)grid;
    if (m < 0 || m >= G->M) return -1;
    for (int i = 0; i < n; ++i) {
        const real p[3] = {(real)xyz[3 * i], (real)xyz[3 * i + 1], (real)xyz[3 * i + 2]};
        real g[3];
        val[i] = trilinear(*G, m, p, grad ? g : nullptr, nullptr, nullptr);
        if (grad) for (int d = 0; d < 3; ++d) grad[3 * i + d] = g[d];
    }
    return 0;
}

int orc_grid_atom(void* grid, const OPar* P, int type, double q, int T, const double* x, double* E, double* g) {
    double fm = 1.0;
    const real p[3] = {(real)x[0], (real)x[1], (real)x[2]};
    real gg[3];
    *E = grid_atom(*(OGrid*)grid, *P, type, (real)q, T, p, gg, &fm);
    for (int d = 0; d < 3; ++d) g[d] = gg[d];
    return 0;
}

int orc_pair_energy(const OPar* P, double c12, double cA, double expA, double qq, double dsco, double d, double* E, double* dEdr) {
    real de;
    *E = pair_energy(*P, (real)c12, (real)cA, (real)expA, (real)qq, (real)dsco, (real)d, &de);
    if (dEdr) *dEdr = de;
    return 0;
}

int orc_score(void* grid, void* lig, const OPar* P, const float* genos, int n, int gstride, double* E, double* terms,
              double* grad, double* margins, double* scales, int nthreads) {
    OGrid* G = (OGrid*)grid;
    OLig* L = (OLig*)lig;
    if (L->T + 2 > G->M) return -1;
    const int Gn = 7 + L->R, D = 6 + L->R;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) {
        std::vector<double> g(Gn);
        for (int d = 0; d < Gn; ++d) g[d] = genos[(size_t)i * gstride + d];
        E[i] = score(*G, *L, *P, g.data(), grad ? grad + (size_t)i * D : nullptr, terms ? terms + 2 * (size_t)i : nullptr,
                     margins ? margins + 2 * (size_t)i : nullptr, scales ? scales + 3 * (size_t)i : nullptr);
    }
    return 0;
}

int orc_score_f64(void* grid, void* lig, const OPar* P, const double* geno, double* E, double* grad) {
    *E = score(*(OGrid*)grid, *(OLig*)lig, *P, geno, grad, nullptr, nullptr);
    return 0;
}

typedef double (*orc_fn)(int n, const double* x, double* grad, void* user);
// generic R^n ADADELTA (Zeiler): x updated in place, f(x_it) recorded before each step
int orc_adadelta_rn(int n, double* x, double rho, double eps, int iters, orc_fn fn, void* user, double* trace) {
    std::vector<double> Eg2(n, 0.0), Ed2(n, 0.0), gr(n), delta(n);
    for (int it = 0; it < iters; ++it) {
        double f = fn(n, x, gr.data(), user);
        if (trace) trace[it] = f;
        adadelta_update(n, gr.data(), Eg2.data(), Ed2.data(), rho, eps, delta.data());
        for (int d = 0; d < n; ++d) x[d] += delta[d];
    }
    return 0;
}

// generic R^n Solis-Wets (R11) on a callback; step = x + sign*delta; x0's value E0 is passed in (carried energy)
struct SwRn : SwFn {
    int n; orc_fn fn; void* user;
    double operator()(const double* x) override { return fn(n, x, nullptr, user); }
    void step(double* x, const double* delta, double sign) override { for (int d = 0; d < n; ++d) x[d] += sign * delta[d]; }
};
int orc_solis_wets_rn(int n, double* x, double* E, const double* amp, const OPar* P, unsigned long long seed, unsigned id, unsigned gen,
                      orc_fn fn, void* user, int* iters, double* rho_out, double* traceE) {
    SwRn f; f.n = n; f.fn = fn; f.user = user;
    return solis_wets(f, n, n, amp, *P, seed, id, gen, x, E, iters, rho_out, traceE);
}
int orc_solis_wets(void* grid, void* lig, const OPar* P, unsigned long long seed, unsigned id, unsigned gen, double* geno, double* E,
                   int* iters, double* rho_out, double* traceE) {
    return solis_wets_dock(*(OGrid*)grid, *(OLig*)lig, *P, seed, id, gen, geno, E, iters, rho_out, traceE);
}

int orc_apply_step(int R, double* x, const double* delta) { apply_step(R, x, delta); return 0; }

int orc_adadelta(void* grid, void* lig, const OPar* P, double* geno, double* E, int* iters, double* traceE, double* traceX) {
    *iters = adadelta_dock(*(OGrid*)grid, *(OLig*)lig, *P, geno, E, traceE, traceX);
    return 0;
}

void orc_philox(const uint32_t* key, const uint32_t* ctr, int n, uint32_t* out) {
    for (int i = 0; i < n; ++i) philox(key, ctr + 4 * (size_t)i, out + 4 * (size_t)i);
}

int orc_ga_init(void* grid, int R, unsigned long long seed, int run, int Pn, double* pop) {
    for (int s = 0; s < Pn; ++s) ga_init_one(*(OGrid*)grid, R, seed, (uint32_t)(run * Pn + s), pop + (size_t)s * (7 + R));
    return 0;
}

int orc_ga_offspring(const OPar* P, int Pn, int R, int run, int gen, unsigned long long seed, const double* pop, const double* E,
                     double* newpop, double* newE, int* dec) {
    ga_offspring(*P, Pn, R, run, gen, seed, pop, E, newpop, newE, dec);
    return 0;
}

int orc_ls_pick(const OPar* P, int Pn, int run, int gen, unsigned long long seed, int* picks) {
    return ls_pick(*P, Pn, run, gen, seed, picks);
}

// full docking: per run best genotype [nrun][7+R], energy, coords (optional), evals, gens; history (optional):
// hist[run][hist_len] best energy of the population after generation 0,1,... (NaN padded)
int orc_dock(void* grid, void* lig, const OPar* P, int nrun, int Pn, long long max_evals, unsigned long long seed,
             double* best_geno, double* best_E, double* best_xyz, long long* evals, int* gens, double* hist, int hist_len,
             int nthreads) {
    OGrid* G = (OGrid*)grid;
    OLig* L = (OLig*)lig;
    if (L->T + 2 > G->M || nrun < 1 || Pn < 2) return -1;
    const int Gn = 7 + L->R;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int run = 0; run < nrun; ++run) {
        std::vector<double> h;
        RunResult r = dock_run(*G, *L, *P, run, Pn, max_evals, seed, hist ? &h : nullptr);
        std::copy(r.best.begin(), r.best.end(), best_geno + (size_t)run * Gn);
        best_E[run] = r.bestE;
        if (best_xyz) {
            std::vector<real> x(3 * L->N);
            pose(*L, r.best.data(), x.data());
            std::copy(x.begin(), x.end(), best_xyz + (size_t)run * 3 * L->N);
        }
        if (evals) evals[run] = r.evals;
        if (gens) gens[run] = r.gens;
        if (hist)
            for (int i = 0; i < hist_len; ++i)
                hist[(size_t)run * hist_len + i] = i < (int)h.size() ? h[i] : std::numeric_limits<double>::quiet_NaN();
    }
    return 0;
}

int orc_real_bytes(void) { return (int)sizeof(real); }

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
