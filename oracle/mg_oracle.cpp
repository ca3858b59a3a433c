// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded fp64 CPU implementation of the
// paper's hot path (arXiv 2509.11831): 5-point discretisation on a locally Cartesian, logically
// unstructured mesh, geometric-multigrid V-cycle with red-black-boundary Gauss-Seidel, fGMRES(m).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
// It shares no code with the CUDA path (paper_2509_11831_b200/csrc) and neither includes the other.
//
// Every function cites the PAPER.md passage it restates ("P:<line>") and, where the paper is silent
// or garbled, the reading of DESIGN.md section 3 ("M*", "D*", "T*", "GS", "C", "V", "K*" rules).
// Parity pins: every function here is pinned by tests/test_oracle_*.py (-m "not gpu"); none is
// "parity unpinned".  Compile: g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC.
// The `#pragma omp` lines are inert in that build (single thread, the arithmetic the pins check).  bench.py's second,
// separately labelled baseline compiles the same file with -fopenmp (grid loops on all host cores, the analogue of the
// paper's OpenMP backend); there the reductions sum in another order, so it is a timing line only.
//
// Conventions: levels are 0-based here (level 0 = the paper's sigma=1, finest).  Every per-level
// vector is in the level's canonical order: ascending (J, I) (rule M7).  User vectors (update/solve)
// are in the caller's point order and are permuted on entry/exit.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

namespace {

enum : uint8_t { INNER = 0, DIRICHLET = 1, NEUMANN = 2 };
enum : uint8_t { RED = 0, BLACK = 1, GUARD = 2 };

static std::string g_err;

// Dense (I,J) -> index lookup over the level's bounding box (+1 ring). -1 = not in the mesh.
struct Lookup {
    int32_t i0 = 0, j0 = 0, ni = 0, nj = 0;
    std::vector<int32_t> a;
    void init(int32_t imin, int32_t imax, int32_t jmin, int32_t jmax) {
        i0 = imin - 2; j0 = jmin - 2; ni = imax - imin + 5; nj = jmax - jmin + 5;
        a.assign((size_t)ni * nj, -1);
    }
    int32_t get(int64_t I, int64_t J) const {
        int64_t x = I - i0, y = J - j0;
        if (x < 0 || y < 0 || x >= ni || y >= nj) return -1;
        return a[(size_t)y * ni + x];
    }
    void set(int32_t I, int32_t J, int32_t v) { a[(size_t)(J - j0) * ni + (I - i0)] = v; }
};

struct Level {
    int64_t n = 0;
    double h = 0;
    std::vector<int32_t> I, J;
    std::vector<uint8_t> kind, colour;
    std::vector<int32_t> nbr;                 // 4n: W, E, S, N   (rule M5)
    // Neumann rows (rule D3): up to 4 non-self nodes
    std::vector<int32_t> ns_idx;              // 4n, -1 = unused
    std::vector<double> ns_w;                 // 4n
    std::vector<double> ns_wself, ns_delta;   // n
    std::vector<int8_t> ns_tn;                // 2n: 2*n^R, 2*n^Z
    std::vector<uint8_t> ns_fallback;         // n
    // transfer tables towards the next COARSER level (empty on the coarsest level)
    std::vector<int32_t> fine9;               // 9 * n_coarse, stored on the FINE level
    std::vector<int32_t> parent;              // 4n: coarse parents of each point of this level
    std::vector<double> parent_w;             // 4n
    std::vector<uint8_t> ptype;               // 0 coincident, 1 R-edge, 2 Z-edge, 3 centre
    std::vector<double> lam, c;
    std::vector<double> xi;                   // the paper's third field (Eq. 3, Eq. 10); 1 unless orc_update3 set it
    Lookup lut;
};

static int64_t floordiv2(int64_t a) { return (a >= 0) ? a / 2 : -((-a + 1) / 2); }

struct Oracle {
    int L = 0;
    std::vector<Level> lev;
    std::vector<int64_t> user2canon;          // user index -> canonical index on level 0
    int nu_pre = 2, nu_post = 2, m = 30, max_iters = 200;
    int gamma = 1;                            // cycle type: 1 V-cycle, 2 W-cycle, 3 F-cycle
    int bc_transfer = 0;                      // 0: rules T2 / T3 (fixed weights, missing points count 0); 1: boundary-aware variant (reading G9)
    bool have_coeffs = false;
    // coarse factorisation
    std::vector<double> lu;
    std::vector<int32_t> piv;
    // dense exact inverse of level 0 (precond_mode 2, tests only)
    std::vector<double> lu0;
    std::vector<int32_t> piv0;
};

// ------------------------------------------------------------------ mesh construction (M1-M7)
static void sort_canonical(std::vector<int32_t>& I, std::vector<int32_t>& J, std::vector<uint8_t>& kind,
                           std::vector<int64_t>* perm_out) {
    size_t n = I.size();
    std::vector<int64_t> p(n);
    for (size_t k = 0; k < n; k++) p[k] = (int64_t)k;
    std::sort(p.begin(), p.end(), [&](int64_t a, int64_t b) {
        if (J[a] != J[b]) return J[a] < J[b];
        return I[a] < I[b];
    });
    std::vector<int32_t> I2(n), J2(n);
    std::vector<uint8_t> k2(n);
    for (size_t k = 0; k < n; k++) { I2[k] = I[p[k]]; J2[k] = J[p[k]]; k2[k] = kind[p[k]]; }
    I.swap(I2); J.swap(J2); kind.swap(k2);
    if (perm_out) {                            // user index -> canonical position
        perm_out->assign(n, 0);
        for (size_t k = 0; k < n; k++) (*perm_out)[p[k]] = (int64_t)k;
    }
}

static void build_lookup(Level& lv) {
    int32_t imin = lv.I[0], imax = lv.I[0], jmin = lv.J[0], jmax = lv.J[0];
    for (int64_t k = 0; k < lv.n; k++) {
        imin = std::min(imin, lv.I[k]); imax = std::max(imax, lv.I[k]);
        jmin = std::min(jmin, lv.J[k]); jmax = std::max(jmax, lv.J[k]);
    }
    lv.lut.init(imin, imax, jmin, jmax);
    for (int64_t k = 0; k < lv.n; k++) lv.lut.set(lv.I[k], lv.J[k], (int32_t)k);
}

// M5 neighbours, M6 colour (red <=> (I+J) even), D3 Neumann stencils (Eq. 12-16).
static void finish_level(Level& lv) {
    const int64_t n = lv.n;
    lv.nbr.assign(4 * n, -1);
    lv.colour.assign(n, GUARD);
    lv.ns_idx.assign(4 * n, -1);
    lv.ns_w.assign(4 * n, 0.0);
    lv.ns_wself.assign(n, 0.0);
    lv.ns_delta.assign(n, 0.0);
    lv.ns_tn.assign(2 * n, 0);
    lv.ns_fallback.assign(n, 0);
    for (int64_t l = 0; l < n; l++) {
        const int32_t I = lv.I[l], J = lv.J[l];
        lv.nbr[4 * l + 0] = lv.lut.get(I - 1, J);
        lv.nbr[4 * l + 1] = lv.lut.get(I + 1, J);
        lv.nbr[4 * l + 2] = lv.lut.get(I, J - 1);
        lv.nbr[4 * l + 3] = lv.lut.get(I, J + 1);
        if (lv.kind[l] == INNER) lv.colour[l] = (((int64_t)I + J) % 2 == 0) ? RED : BLACK;
    }
    // Eq. 12: twice the level-set function, 2 = inner, 1 = boundary, 0 = not in mesh
    auto psi2 = [&](int32_t idx) -> int { return idx < 0 ? 0 : (lv.kind[idx] == INNER ? 2 : 1); };
    for (int64_t l = 0; l < n; l++) {
        if (lv.kind[l] != NEUMANN) continue;
        const int32_t I = lv.I[l], J = lv.J[l];
        // Eq. 13, stored doubled: tnR = 2 n^R in {-2..2}
        const int tnR = psi2(lv.nbr[4 * l + 1]) - psi2(lv.nbr[4 * l + 0]);
        const int tnZ = psi2(lv.nbr[4 * l + 3]) - psi2(lv.nbr[4 * l + 2]);
        lv.ns_tn[2 * l] = (int8_t)tnR; lv.ns_tn[2 * l + 1] = (int8_t)tnZ;
        // per-axis offsets/weights: integer n -> {n}; half-integer n -> {0, 2n} with 1/2, 1/2 (Eq. 14/15)
        int offR[2], offZ[2], nR, nZ; double wR[2], wZ[2];
        if (tnR % 2 == 0) { nR = 1; offR[0] = tnR / 2; wR[0] = 1.0; }
        else { nR = 2; offR[0] = 0; offR[1] = tnR; wR[0] = wR[1] = 0.5; }
        if (tnZ % 2 == 0) { nZ = 1; offZ[0] = tnZ / 2; wZ[0] = 1.0; }
        else { nZ = 2; offZ[0] = 0; offZ[1] = tnZ; wZ[0] = wZ[1] = 0.5; }
        bool fallback = (tnR == 0 && tnZ == 0);
        int cnt = 0; double wself = 0.0; int32_t idx[4]; double w[4];
        if (!fallback) {
            for (int b = 0; b < nZ && !fallback; b++)
                for (int a = 0; a < nR; a++) {
                    const double ww = wR[a] * wZ[b];
                    if (offR[a] == 0 && offZ[b] == 0) { wself += ww; continue; }
                    const int32_t q = lv.lut.get(I + offR[a], J + offZ[b]);
                    if (q < 0 || lv.kind[q] != INNER) { fallback = true; break; }   // P:123 inner only
                    idx[cnt] = q; w[cnt] = ww; cnt++;
                }
        }
        if (fallback) {
            // reading G7: mean of the inner 4-neighbours, delta = h
            cnt = 0; wself = 0.0;
            for (int d = 0; d < 4; d++) {
                const int32_t q = lv.nbr[4 * l + d];
                if (q >= 0 && lv.kind[q] == INNER) idx[cnt++] = q;
            }
            for (int k = 0; k < cnt; k++) w[k] = 1.0 / cnt;
            lv.ns_delta[l] = lv.h;
            lv.ns_fallback[l] = 1;
        } else {
            lv.ns_delta[l] = lv.h * std::sqrt(0.25 * (double)(tnR * tnR + tnZ * tnZ));   // Eq. 16
        }
        lv.ns_wself[l] = wself;
        for (int k = 0; k < cnt; k++) { lv.ns_idx[4 * l + k] = idx[k]; lv.ns_w[4 * l + k] = w[k]; }
    }
}

// M3 coarsening + M2 guards + M4 type inheritance.  Returns false if the coarse inner set is empty.
static bool coarsen(const Level& f, Level& c) {
    std::vector<int32_t> I, J; std::vector<uint8_t> kind;
    for (int64_t l = 0; l < f.n; l++)
        if (f.kind[l] == INNER && (f.I[l] % 2 == 0) && (f.J[l] % 2 == 0)) {
            I.push_back((int32_t)floordiv2(f.I[l])); J.push_back((int32_t)floordiv2(f.J[l])); kind.push_back(INNER);
        }
    if (I.empty()) return false;
    const size_t n_in = I.size();
    Level tmp; tmp.n = (int64_t)n_in; tmp.I = I; tmp.J = J; tmp.kind = kind;
    build_lookup(tmp);                                  // inner-only lookup
    static const int dI[4] = {-1, 1, 0, 0}, dJ[4] = {0, 0, -1, 1};
    // guards: non-inner 4-neighbours of coarse inner points (dedupe through a second lookup)
    Lookup seen; seen.init(tmp.lut.i0 + 2, tmp.lut.i0 + tmp.lut.ni - 3, tmp.lut.j0 + 2, tmp.lut.j0 + tmp.lut.nj - 3);
    for (size_t q = 0; q < n_in; q++)
        for (int d = 0; d < 4; d++) {
            const int32_t gi = I[q] + dI[d], gj = J[q] + dJ[d];
            if (tmp.lut.get(gi, gj) >= 0) continue;
            if (seen.get(gi, gj) >= 0) continue;
            seen.set(gi, gj, 1);
            // M4: candidates over all coarse inner 4-neighbours of g; Dirichlet wins
            bool any_dir = false;
            for (int e = 0; e < 4; e++) {
                const int32_t qi = gi + dI[e], qj = gj + dJ[e];
                if (tmp.lut.get(qi, qj) < 0) continue;
                const int32_t mi = gi + qi, mj = gj + qj;           // fine-lattice midpoint of g and q
                const int32_t mid = f.lut.get(mi, mj);
                uint8_t cand;
                if (mid >= 0 && f.kind[mid] == INNER) {
                    const int32_t gf = f.lut.get(2 * gi, 2 * gj);   // g itself is a fine guard
                    cand = f.kind[gf];
                } else {
                    cand = f.kind[mid];                             // the midpoint is a fine guard
                }
                if (cand == DIRICHLET) any_dir = true;
            }
            I.push_back(gi); J.push_back(gj); kind.push_back(any_dir ? DIRICHLET : NEUMANN);
        }
    c.I = I; c.J = J; c.kind = kind; c.n = (int64_t)I.size(); c.h = 2.0 * f.h;   // reading G2 of P:151
    sort_canonical(c.I, c.J, c.kind, nullptr);
    build_lookup(c);
    finish_level(c);
    return true;
}

// Transfer tables between f (fine) and c (next coarser): T1 stencils, Fig. 3.
static void build_transfers(Level& f, const Level& c) {
    f.fine9.assign(9 * c.n, -1);
    for (int64_t q = 0; q < c.n; q++)
        for (int dy = -1; dy <= 1; dy++)
            for (int dx = -1; dx <= 1; dx++)
                f.fine9[9 * q + 3 * (dy + 1) + (dx + 1)] = f.lut.get(2 * (int64_t)c.I[q] + dx, 2 * (int64_t)c.J[q] + dy);
    f.parent.assign(4 * f.n, -1);
    f.parent_w.assign(4 * f.n, 0.0);
    f.ptype.assign(f.n, 0);
    for (int64_t l = 0; l < f.n; l++) {
        const int64_t I = f.I[l], J = f.J[l];
        const bool oi = (I % 2 != 0), oj = (J % 2 != 0);
        const int64_t Il = floordiv2(I), Jl = floordiv2(J);       // lower coarse index
        int cnt = 0;
        auto add = [&](int64_t ci, int64_t cj, double w) {
            f.parent[4 * l + cnt] = c.lut.get(ci, cj); f.parent_w[4 * l + cnt] = w; cnt++;
        };
        if (!oi && !oj) { f.ptype[l] = 0; add(Il, Jl, 1.0); }
        else if (oi && !oj) { f.ptype[l] = 1; add(Il, Jl, 0.5); add(Il + 1, Jl, 0.5); }
        else if (!oi && oj) { f.ptype[l] = 2; add(Il, Jl, 0.5); add(Il, Jl + 1, 0.5); }
        else { f.ptype[l] = 3; add(Il, Jl, 0.25); add(Il + 1, Jl, 0.25); add(Il, Jl + 1, 0.25); add(Il + 1, Jl + 1, 0.25); }
    }
}

// ------------------------------------------------------------------ discretisation (D1-D3)
// Row l of A^sigma applied to x.  Inner: Eq. 10 with the 1/h^2 restored (reading G1);
// Dirichlet: Eq. 11; Neumann: Eq. 16 with phi^N of rule D3.
static inline double row_apply(const Level& lv, int64_t l, const double* x) {
    if (lv.kind[l] == INNER) {
        // Eq. 10: the bracket carries xi_{i,j}/2 of the ROW's own point; 1/h^2 restored (reading G1)
        const double kappa = 1.0 / (2.0 * lv.h * lv.h) * lv.xi[l];
        const int32_t* nb = &lv.nbr[4 * l];
        const double cl = lv.c[l];
        const double aW = kappa * (cl + lv.c[nb[0]]);
        const double aE = kappa * (cl + lv.c[nb[1]]);
        const double aS = kappa * (cl + lv.c[nb[2]]);
        const double aN = kappa * (cl + lv.c[nb[3]]);
        // same row as Eq. 10, evaluated in difference form (rule D1): lam x_l + sum a_nb (x_l - x_nb).
        // Algebraically identical to a_ll x_l - sum a_nb x_nb, but free of the O(eps |a_ll x_l|)
        // cancellation error that otherwise puts the attainable residual above 1e-10 at h ~ 5e-4.
        const double xl = x[l];
        return lv.lam[l] * xl + aW * (xl - x[nb[0]]) + aE * (xl - x[nb[1]]) + aS * (xl - x[nb[2]]) + aN * (xl - x[nb[3]]);
    }
    if (lv.kind[l] == DIRICHLET) return x[l];
    double phiN = lv.ns_wself[l] * x[l];
    for (int k = 0; k < 4; k++) {
        const int32_t q = lv.ns_idx[4 * l + k];
        if (q >= 0) phiN += lv.ns_w[4 * l + k] * x[q];
    }
    return (phiN - x[l]) / lv.ns_delta[l];
}

static void apply(const Level& lv, const double* x, double* y) {
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < lv.n; l++) y[l] = row_apply(lv, l, x);
}

// One group of gauss_seidel_rbb: group 0 red inner, 1 black inner, 2 boundary.
static void gs_group(const Level& lv, double* x, const double* b, int group) {
    const double kappa0 = 1.0 / (2.0 * lv.h * lv.h);
#pragma omp parallel for schedule(static)      // the points of one group are independent
    for (int64_t l = 0; l < lv.n; l++) {
        if (lv.colour[l] != group) continue;
        if (lv.kind[l] == INNER) {
            const double kappa = kappa0 * lv.xi[l];                  // xi_{i,j}/2 of Eq. 10
            const int32_t* nb = &lv.nbr[4 * l];
            const double cl = lv.c[l];
            const double aW = kappa * (cl + lv.c[nb[0]]);
            const double aE = kappa * (cl + lv.c[nb[1]]);
            const double aS = kappa * (cl + lv.c[nb[2]]);
            const double aN = kappa * (cl + lv.c[nb[3]]);
            const double all = lv.lam[l] + aW + aE + aS + aN;
            x[l] = (b[l] + aW * x[nb[0]] + aE * x[nb[1]] + aS * x[nb[2]] + aN * x[nb[3]]) / all;
        } else if (lv.kind[l] == DIRICHLET) {
            x[l] = b[l];                                             // Eq. 11
        } else {                                                     // Eq. 16 solved for x_l
            double s = 0.0;
            for (int k = 0; k < 4; k++) {
                const int32_t q = lv.ns_idx[4 * l + k];
                if (q >= 0) s += lv.ns_w[4 * l + k] * x[q];
            }
            x[l] = (s - lv.ns_delta[l] * b[l]) / (1.0 - lv.ns_wself[l]);
        }
    }
}

static void gs_sweep(const Level& lv, double* x, const double* b) {
    gs_group(lv, x, b, RED); gs_group(lv, x, b, BLACK); gs_group(lv, x, b, GUARD);
}

// ------------------------------------------------------------------ transfers (T1-T4)
static const double FW[9] = {1.0 / 16, 2.0 / 16, 1.0 / 16, 2.0 / 16, 4.0 / 16, 2.0 / 16, 1.0 / 16, 2.0 / 16, 1.0 / 16};

// T2: full-weighting restriction of the defect; fine guards/absent count 0;
// coarse guard rows are reset to 0 ("boundary values can explicitly be reset").
// bc_mode 1 (experiment of reading G9, "stencil points may be missing"): where the 3 x 3 fine neighbourhood of the
// coarse point touches a NEUMANN guard, the weights of the fine inner points present are renormalised to sum 1 (at a
// Dirichlet boundary the missing defects really are 0, at a Neumann boundary they are not).
static void restrict_defect(const Level& f, const Level& c, const double* df, double* dc, int bc_mode = 0) {
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < c.n; q++) {
        if (c.kind[q] != INNER) { dc[q] = 0.0; continue; }
        double s = 0.0, w = 0.0;
        bool neu = false;
        for (int k = 0; k < 9; k++) {
            const int32_t l = f.fine9[9 * q + k];
            if (l >= 0 && f.kind[l] == INNER) { s += FW[k] * df[l]; w += FW[k]; }
            if (l >= 0 && f.kind[l] == NEUMANN) neu = true;
        }
        dc[q] = (bc_mode == 1 && neu && w > 0.0) ? s / w : s;
    }
}

// T3: e = P e_c on fine inner points (bilinear, absent parents count 0), set_bnds_hom on fine guards
// (homogeneous Eq. 11/16), then x <- x - e.
// bc_mode 1 (reading G9 experiment): a fine inner point with an absent parent and a Neumann guard among its 4-neighbours
// interpolates from the parents present with weights renormalised to sum 1 (zero-filling is exact only for Dirichlet data).
static void prolong_correct(const Level& f, const double* ec, double* x, std::vector<double>& e, int bc_mode = 0) {
    e.assign(f.n, 0.0);
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < f.n; l++) {
        if (f.kind[l] != INNER) continue;
        double s = 0.0, w = 0.0, wall = 0.0;
        for (int k = 0; k < 4; k++) {
            const int32_t p = f.parent[4 * l + k];
            wall += f.parent_w[4 * l + k];
            if (p >= 0) { s += f.parent_w[4 * l + k] * ec[p]; w += f.parent_w[4 * l + k]; }
        }
        if (bc_mode == 1 && w > 0.0 && w < wall) {
            bool neu = false;
            for (int d = 0; d < 4; d++) { const int32_t q = f.nbr[4 * l + d]; if (q >= 0 && f.kind[q] == NEUMANN) neu = true; }
            if (neu) s *= wall / w;
        }
        e[l] = s;
    }
    for (int64_t l = 0; l < f.n; l++) {
        if (f.kind[l] == DIRICHLET) e[l] = 0.0;
        else if (f.kind[l] == NEUMANN) {
            double s = 0.0;
            for (int k = 0; k < 4; k++) {
                const int32_t q = f.ns_idx[4 * l + k];
                if (q >= 0) s += f.ns_w[4 * l + k] * e[q];
            }
            e[l] = s / (1.0 - f.ns_wself[l]);
        }
    }
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < f.n; l++) x[l] -= e[l];
}

// T4: coefficient restriction (P:153 last sentence): full weighting over the fine points present
// in the mesh, renormalised by the weights present.
static void restrict_coeff(const Level& f, const Level& c, const double* vf, double* vc) {
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < c.n; q++) {
        double s = 0.0, w = 0.0;
        for (int k = 0; k < 9; k++) {
            const int32_t l = f.fine9[9 * q + k];
            if (l >= 0) { s += FW[k] * vf[l]; w += FW[k]; }
        }
        vc[q] = s / w;
    }
}

// ------------------------------------------------------------------ dense LU (rule C)
static void assemble_dense(const Level& lv, std::vector<double>& A) {
    const int64_t n = lv.n;
    A.assign((size_t)n * n, 0.0);
    std::vector<double> e(n, 0.0), col(n);
    for (int64_t k = 0; k < n; k++) {
        e[k] = 1.0; apply(lv, e.data(), col.data()); e[k] = 0.0;
        for (int64_t r = 0; r < n; r++) A[(size_t)r * n + k] = col[r];
    }
}

static bool lu_factor(std::vector<double>& A, std::vector<int32_t>& piv, int64_t n) {
    piv.assign(n, 0);
    for (int64_t k = 0; k < n; k++) {
        int64_t p = k; double best = std::fabs(A[(size_t)k * n + k]);
        for (int64_t r = k + 1; r < n; r++) {
            const double v = std::fabs(A[(size_t)r * n + k]);
            if (v > best) { best = v; p = r; }                       // first max wins ties
        }
        if (best == 0.0) return false;
        piv[k] = (int32_t)p;
        if (p != k) for (int64_t cidx = 0; cidx < n; cidx++) std::swap(A[(size_t)k * n + cidx], A[(size_t)p * n + cidx]);
        const double d = A[(size_t)k * n + k];
        for (int64_t r = k + 1; r < n; r++) {
            const double fct = A[(size_t)r * n + k] / d;
            A[(size_t)r * n + k] = fct;
            if (fct != 0.0) for (int64_t cidx = k + 1; cidx < n; cidx++) A[(size_t)r * n + cidx] -= fct * A[(size_t)k * n + cidx];
        }
    }
    return true;
}

static void lu_solve(const std::vector<double>& A, const std::vector<int32_t>& piv, int64_t n, const double* b, double* x) {
    std::vector<double> y(b, b + n);
    for (int64_t k = 0; k < n; k++) std::swap(y[k], y[piv[k]]);    // P b (whole rows were swapped in lu_factor)
    for (int64_t k = 0; k < n; k++)
        for (int64_t r = k + 1; r < n; r++) y[r] -= A[(size_t)r * n + k] * y[k];
    for (int64_t k = n - 1; k >= 0; k--) {
        double s = y[k];
        for (int64_t cidx = k + 1; cidx < n; cidx++) s -= A[(size_t)k * n + cidx] * y[cidx];
        y[k] = s / A[(size_t)k * n + k];
    }
    std::memcpy(x, y.data(), sizeof(double) * n);
}

// ------------------------------------------------------------------ mg_cycle
// kind: 1 = V (gamma = 1), 2 = W (gamma = 2); 3 = F: the next coarser level is visited twice like gamma = 2,
// first by an F-cycle, then by a V-cycle (the paper names F-cycles at P:258 and defers to its ref. [33]).
static void mg_cycle(Oracle& o, int s, double* x, const double* b, int kind) {
    Level& lv = o.lev[s];
    if (s == o.L - 1) { lu_solve(o.lu, o.piv, lv.n, b, x); return; }
    for (int k = 0; k < o.nu_pre; k++) gs_sweep(lv, x, b);
    std::vector<double> d(lv.n);
    apply(lv, x, d.data());
    for (int64_t l = 0; l < lv.n; l++) d[l] = d[l] - b[l];                   // P:183 d = A x - b
    Level& cv = o.lev[s + 1];
    std::vector<double> dc(cv.n), ec(cv.n, 0.0);                             // P:186 e = 0
    restrict_defect(lv, cv, d.data(), dc.data(), o.bc_transfer);
    if (kind == 3) {
        mg_cycle(o, s + 1, ec.data(), dc.data(), 3);
        mg_cycle(o, s + 1, ec.data(), dc.data(), 1);
    } else {
        for (int g = 0; g < kind; g++) mg_cycle(o, s + 1, ec.data(), dc.data(), kind);   // gamma visits, e carried over
    }
    std::vector<double> e;
    prolong_correct(lv, ec.data(), x, e, o.bc_transfer);
    for (int k = 0; k < o.nu_post; k++) gs_sweep(lv, x, b);
}

static double dot(const double* a, const double* b, int64_t n) {
    double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (int64_t k = 0; k < n; k++) s += a[k] * b[k];
    return s;
}

}  // namespace

// ====================================================================== C interface (ctypes)
extern "C" {

const char* orc_last_error() { return g_err.c_str(); }

void orc_destroy(void* h) { delete (Oracle*)h; }

// levels = 0 -> auto (rule M8).  Returns NULL on invalid input (orc_last_error says why).
void* orc_create(int64_t n, const int32_t* i, const int32_t* j, const uint8_t* kind, double h,
                 int levels, int nu_pre, int nu_post, int m, int max_iters) {
    g_err.clear();
    if (n <= 0 || !i || !j || !kind || !(h > 0.0)) { g_err = "invalid argument"; return nullptr; }
    Oracle* o = new Oracle();
    o->nu_pre = nu_pre; o->nu_post = nu_post; o->m = m; o->max_iters = max_iters;
    o->lev.reserve(64);
    o->lev.emplace_back();
    Level& l0 = o->lev[0];
    l0.n = n; l0.h = h;
    l0.I.assign(i, i + n); l0.J.assign(j, j + n); l0.kind.assign(kind, kind + n);
    for (int64_t k = 0; k < n; k++) if (kind[k] > 2) { g_err = "kind out of range"; delete o; return nullptr; }
    sort_canonical(l0.I, l0.J, l0.kind, &o->user2canon);
    for (int64_t k = 1; k < n; k++)
        if (l0.I[k] == l0.I[k - 1] && l0.J[k] == l0.J[k - 1]) { g_err = "duplicate (i,j)"; delete o; return nullptr; }
    build_lookup(l0);
    // M2 validation: inner points have 4 neighbours; guards are exactly the 4-adjacent non-inner points
    static const int dI[4] = {-1, 1, 0, 0}, dJ[4] = {0, 0, -1, 1};
    for (int64_t k = 0; k < n; k++) {
        bool has_inner = false;
        for (int d = 0; d < 4; d++) {
            const int32_t q = l0.lut.get(l0.I[k] + dI[d], l0.J[k] + dJ[d]);
            if (l0.kind[k] == INNER && q < 0) { g_err = "inner point lacks a neighbour"; delete o; return nullptr; }
            if (q >= 0 && l0.kind[q] == INNER) has_inner = true;
        }
        if (l0.kind[k] != INNER && !has_inner) { g_err = "guard without inner 4-neighbour"; delete o; return nullptr; }
    }
    finish_level(l0);
    // M8: level count
    const int want = levels > 0 ? levels : 64;
    while ((int)o->lev.size() < want) {
        Level& f = o->lev.back();
        if (levels <= 0) {
            int32_t imin = f.I[0], imax = f.I[0], jmin = f.J[0], jmax = f.J[0];
            for (int64_t k = 0; k < f.n; k++) {
                imin = std::min(imin, f.I[k]); imax = std::max(imax, f.I[k]);
                jmin = std::min(jmin, f.J[k]); jmax = std::max(jmax, f.J[k]);
            }
            if (std::max(imax - imin + 1, jmax - jmin + 1) <= 9) break;
        }
        Level c;
        if (!coarsen(f, c)) break;
        if (levels <= 0) {
            int64_t nin = 0;
            for (int64_t k = 0; k < c.n; k++) nin += (c.kind[k] == INNER);
            if (nin < 16) break;
        }
        o->lev.push_back(std::move(c));
        build_transfers(o->lev[o->lev.size() - 2], o->lev.back());
    }
    o->L = (int)o->lev.size();
    for (auto& lv : o->lev) { lv.lam.assign(lv.n, 0.0); lv.c.assign(lv.n, 0.0); lv.xi.assign(lv.n, 1.0); }
    return o;
}

// cycle type: gamma of P:187-189 (1 = V, 2 = W) or 3 = F-cycle; default 1
void orc_set_gamma(void* h, int gamma) { ((Oracle*)h)->gamma = (gamma < 1 || gamma > 3) ? 1 : gamma; }

// 1: boundary-aware transfers inside the cycle (reading G9 experiment; the single-step entry points keep rules T2 / T3)
void orc_set_bc_transfer(void* h, int mode) { ((Oracle*)h)->bc_transfer = mode == 1 ? 1 : 0; }

int orc_num_levels(void* h) { return ((Oracle*)h)->L; }
int64_t orc_level_n(void* h, int s) { return ((Oracle*)h)->lev[s].n; }
double orc_level_h(void* h, int s) { return ((Oracle*)h)->lev[s].h; }

// user index -> canonical level-0 index
void orc_user_perm(void* h, int64_t* out) {
    Oracle* o = (Oracle*)h;
    std::memcpy(out, o->user2canon.data(), sizeof(int64_t) * o->user2canon.size());
}

// any pointer may be NULL
void orc_level_arrays(void* h, int s, int32_t* I, int32_t* J, uint8_t* kind, uint8_t* colour, int32_t* nbr,
                      int32_t* ns_idx, double* ns_w, double* ns_wself, double* ns_delta, int8_t* ns_tn,
                      uint8_t* ns_fallback) {
    Level& lv = ((Oracle*)h)->lev[s];
    const int64_t n = lv.n;
    if (I) std::memcpy(I, lv.I.data(), 4 * n);
    if (J) std::memcpy(J, lv.J.data(), 4 * n);
    if (kind) std::memcpy(kind, lv.kind.data(), n);
    if (colour) std::memcpy(colour, lv.colour.data(), n);
    if (nbr) std::memcpy(nbr, lv.nbr.data(), 16 * n);
    if (ns_idx) std::memcpy(ns_idx, lv.ns_idx.data(), 16 * n);
    if (ns_w) std::memcpy(ns_w, lv.ns_w.data(), 32 * n);
    if (ns_wself) std::memcpy(ns_wself, lv.ns_wself.data(), 8 * n);
    if (ns_delta) std::memcpy(ns_delta, lv.ns_delta.data(), 8 * n);
    if (ns_tn) std::memcpy(ns_tn, lv.ns_tn.data(), 2 * n);
    if (ns_fallback) std::memcpy(ns_fallback, lv.ns_fallback.data(), n);
}

// tables between level s (fine) and s+1: fine9 [9*n_{s+1}], parent [4*n_s], parent_w [4*n_s], ptype [n_s]
void orc_transfer_tables(void* h, int s, int32_t* fine9, int32_t* parent, double* parent_w, uint8_t* ptype) {
    Oracle* o = (Oracle*)h;
    Level& f = o->lev[s];
    if (fine9) std::memcpy(fine9, f.fine9.data(), 4 * f.fine9.size());
    if (parent) std::memcpy(parent, f.parent.data(), 4 * f.parent.size());
    if (parent_w) std::memcpy(parent_w, f.parent_w.data(), 8 * f.parent_w.size());
    if (ptype) std::memcpy(ptype, f.ptype.data(), f.ptype.size());
}

// "update": coefficients in USER order on all points; T4 to all coarser levels;
// LU-factorise the coarsest operator.  Returns 0, or -1 if a coefficient is not admissible (c <= 0 or non-finite),
// -2 if the coarsest matrix is singular.
// xi == NULL: the two-field form of BASELINE.json (paper xi = 1).  Otherwise xi is the paper's third field
// (Eq. 3; Eq. 10), grid-transferred like lambda and c ("lambda, xi, c") and required > 0.
int orc_update3(void* h, const double* lam, const double* xi, const double* c) {
    Oracle* o = (Oracle*)h;
    Level& l0 = o->lev[0];
    for (int64_t k = 0; k < l0.n; k++) {
        // c > 0 is required; lambda >= 0 is only the paper's sufficient condition for positive definiteness and its own
        // verification case has lambda = r sin(theta) of both signs (Eq. 21), so lambda is only required to be finite
        if (!(c[k] > 0.0) || !std::isfinite(c[k]) || !std::isfinite(lam[k])) { g_err = "need c>0 and finite lambda"; return -1; }
        if (xi && (!(xi[k] > 0.0) || !std::isfinite(xi[k]))) { g_err = "need xi>0"; return -1; }
        l0.lam[o->user2canon[k]] = lam[k];
        l0.c[o->user2canon[k]] = c[k];
        l0.xi[o->user2canon[k]] = xi ? xi[k] : 1.0;
    }
    for (int s = 0; s + 1 < o->L; s++) {
        restrict_coeff(o->lev[s], o->lev[s + 1], o->lev[s].lam.data(), o->lev[s + 1].lam.data());
        restrict_coeff(o->lev[s], o->lev[s + 1], o->lev[s].c.data(), o->lev[s + 1].c.data());
        if (xi) restrict_coeff(o->lev[s], o->lev[s + 1], o->lev[s].xi.data(), o->lev[s + 1].xi.data());
        else o->lev[s + 1].xi.assign(o->lev[s + 1].n, 1.0);
    }
    assemble_dense(o->lev[o->L - 1], o->lu);
    if (!lu_factor(o->lu, o->piv, o->lev[o->L - 1].n)) { g_err = "singular coarsest operator"; return -2; }
    o->have_coeffs = true;
    o->lu0.clear();
    return 0;
}

int orc_update(void* h, const double* lam, const double* c) { return orc_update3(h, lam, nullptr, c); }

void orc_level_xi(void* h, int s, double* xi) {
    Level& lv = ((Oracle*)h)->lev[s];
    std::memcpy(xi, lv.xi.data(), 8 * lv.n);
}

void orc_level_coeffs(void* h, int s, double* lam, double* c) {
    Level& lv = ((Oracle*)h)->lev[s];
    if (lam) std::memcpy(lam, lv.lam.data(), 8 * lv.n);
    if (c) std::memcpy(c, lv.c.data(), 8 * lv.n);
}

// ---- single applications, level vectors in canonical order
void orc_apply(void* h, int s, const double* x, double* y) { apply(((Oracle*)h)->lev[s], x, y); }
void orc_smooth(void* h, int s, double* x, const double* b, int sweeps) {
    for (int k = 0; k < sweeps; k++) gs_sweep(((Oracle*)h)->lev[s], x, b);
}
void orc_smooth_group(void* h, int s, double* x, const double* b, int group) { gs_group(((Oracle*)h)->lev[s], x, b, group); }
void orc_restrict(void* h, int s, const double* dfine, double* dcoarse) {
    Oracle* o = (Oracle*)h; restrict_defect(o->lev[s], o->lev[s + 1], dfine, dcoarse);
}
void orc_prolong_correct(void* h, int s, const double* ecoarse, double* xfine) {
    Oracle* o = (Oracle*)h; std::vector<double> e; prolong_correct(o->lev[s], ecoarse, xfine, e);
}
void orc_restrict_coeff(void* h, int s, const double* vfine, double* vcoarse) {
    Oracle* o = (Oracle*)h; restrict_coeff(o->lev[s], o->lev[s + 1], vfine, vcoarse);
}
void orc_coarse_solve(void* h, const double* b, double* x) {
    Oracle* o = (Oracle*)h; lu_solve(o->lu, o->piv, o->lev[o->L - 1].n, b, x);
}
void orc_cycle(void* h, int s, double* x, const double* b) { mg_cycle(*(Oracle*)h, s, x, b, ((Oracle*)h)->gamma); }

// fGMRES(m) — Saad's flexible GMRES ([12],[29]), rules K1-K5; stop on Eq. 23.
// Vectors f, x0, x in USER order.  precond: 0 = one V-cycle from zero (G16), 1 = identity,
// 2 = dense exact inverse of A (tests only, small n).
// Optional debug dumps of the FIRST restart cycle (canonical order): V [(m+1) x n], Z [m x n],
// H [(m+1) x m] (raw Hessenberg, row-major), ncols.  hist[k] = |g_{k+1}|/||b|| after iteration k+1.
// Returns 0 converged, 1 max_iters reached, 2 breakdown, <0 error.
int orc_solve_ex(void* h, const double* f_user, const double* x0_user, double* x_user, double rtol, int precond,
                 int* iters_out, double* relres_out, double* hist, double* Vd, double* Zd, double* Hd, int* ncols) {
    Oracle* o = (Oracle*)h;
    if (!o->have_coeffs) { g_err = "solve before update"; return -3; }
    Level& lv = o->lev[0];
    const int64_t n = lv.n; const int m = o->m;
    std::vector<double> b(n), x(n), r(n), w(n);
    for (int64_t k = 0; k < n; k++) { b[o->user2canon[k]] = f_user[k]; x[o->user2canon[k]] = x0_user[k]; }
    if (precond == 2 && o->lu0.empty()) { assemble_dense(lv, o->lu0); if (!lu_factor(o->lu0, o->piv0, n)) return -2; }
    int iters = 0, status = 1; double relres = 0.0; bool first_cycle = true;
    const double bn = std::sqrt(dot(b.data(), b.data(), n));                       // K1
    auto finish = [&](int st) {
        for (int64_t k = 0; k < n; k++) x_user[k] = x[o->user2canon[k]];
        if (iters_out) *iters_out = iters;
        if (relres_out) *relres_out = relres;
        return st;
    };
    if (ncols) *ncols = 0;
    if (bn == 0.0) { std::fill(x.begin(), x.end(), 0.0); return finish(0); }
    std::vector<std::vector<double>> V(m + 1, std::vector<double>(n)), Z(m, std::vector<double>(n));
    std::vector<double> H((size_t)(m + 1) * m, 0.0), Hraw((size_t)(m + 1) * m, 0.0), g(m + 1), cs(m), sn(m), y(m);
    while (true) {
        apply(lv, x.data(), r.data());
        for (int64_t k = 0; k < n; k++) r[k] = b[k] - r[k];                        // D4 r = b - A x
        const double beta = std::sqrt(dot(r.data(), r.data(), n));
        relres = beta / bn;
        if (relres < rtol) { status = 0; break; }                                  // K1 / K5
        if (iters >= o->max_iters) { status = 1; break; }
        for (int64_t k = 0; k < n; k++) V[0][k] = r[k] / beta;                     // K2
        std::fill(g.begin(), g.end(), 0.0); g[0] = beta;
        std::fill(H.begin(), H.end(), 0.0);
        int jdone = 0; bool breakdown = false;
        for (int j = 0; j < m && iters < o->max_iters; j++) {
            if (precond == 0) { std::fill(Z[j].begin(), Z[j].end(), 0.0); mg_cycle(*o, 0, Z[j].data(), V[j].data(), o->gamma); }
            else if (precond == 1) Z[j] = V[j];
            else lu_solve(o->lu0, o->piv0, n, V[j].data(), Z[j].data());
            apply(lv, Z[j].data(), w.data());
            // modified Gram-Schmidt, applied twice (reorthogonalisation, rule K2): the second pass keeps
            // V orthogonal to working precision, so the iteration count does not depend on how the
            // orthogonalisation rounds (identical counts across backends)
            for (int pass = 0; pass < 2; pass++)
                for (int i = 0; i <= j; i++) {
                    const double hij = dot(w.data(), V[i].data(), n);
                    H[(size_t)i * m + j] += hij;
                    {
                        const double* vi = V[i].data();
#pragma omp parallel for schedule(static)
                        for (int64_t k = 0; k < n; k++) w[k] -= hij * vi[k];
                    }
                }
            const double hn = std::sqrt(dot(w.data(), w.data(), n));
            H[(size_t)(j + 1) * m + j] = hn;
            if (first_cycle) for (int i = 0; i <= j + 1; i++) Hraw[(size_t)i * m + j] = H[(size_t)i * m + j];
            for (int i = 0; i < j; i++) {                                          // previous rotations
                const double t = cs[i] * H[(size_t)i * m + j] + sn[i] * H[(size_t)(i + 1) * m + j];
                H[(size_t)(i + 1) * m + j] = -sn[i] * H[(size_t)i * m + j] + cs[i] * H[(size_t)(i + 1) * m + j];
                H[(size_t)i * m + j] = t;
            }
            const double rho = std::hypot(H[(size_t)j * m + j], hn);
            cs[j] = H[(size_t)j * m + j] / rho; sn[j] = hn / rho;
            H[(size_t)j * m + j] = rho; H[(size_t)(j + 1) * m + j] = 0.0;
            g[j + 1] = -sn[j] * g[j]; g[j] = cs[j] * g[j];
            iters++; jdone = j + 1;
            if (hist) hist[iters - 1] = std::fabs(g[j + 1]) / bn;
            if (std::fabs(g[j + 1]) / bn < rtol) break;                            // K3, Eq. 23
            if (hn == 0.0) { breakdown = true; break; }
            for (int64_t k = 0; k < n; k++) V[j + 1][k] = w[k] / hn;
        }
        for (int i = jdone - 1; i >= 0; i--) {                                     // K4: R y = g
            double s = g[i];
            for (int k = i + 1; k < jdone; k++) s -= H[(size_t)i * m + k] * y[k];
            y[i] = s / H[(size_t)i * m + i];
        }
        for (int i = 0; i < jdone; i++)
            {
                const double* zi = Z[i].data();
                const double yi = y[i];
#pragma omp parallel for schedule(static)
                for (int64_t k = 0; k < n; k++) x[k] += yi * zi[k];
            }
        if (first_cycle) {
            if (ncols) *ncols = jdone;
            if (Vd) for (int i = 0; i <= jdone && i <= m; i++) std::memcpy(Vd + (size_t)i * n, V[i].data(), 8 * n);
            if (Zd) for (int i = 0; i < jdone; i++) std::memcpy(Zd + (size_t)i * n, Z[i].data(), 8 * n);
            if (Hd) std::memcpy(Hd, Hraw.data(), 8 * Hraw.size());
            first_cycle = false;
        }
        if (breakdown) {
            apply(lv, x.data(), r.data());
            for (int64_t k = 0; k < n; k++) r[k] = b[k] - r[k];
            relres = std::sqrt(dot(r.data(), r.data(), n)) / bn;
            status = relres < rtol ? 0 : 2;
            break;
        }
    }                                                                              // K5: loop = restart
    return finish(status);
}

int orc_solve(void* h, const double* f, const double* x0, double* x, double rtol, int* iters, double* relres) {
    return orc_solve_ex(h, f, x0, x, rtol, 0, iters, relres, nullptr, nullptr, nullptr, nullptr, nullptr);
}

// BiCGStab (van der Vorst) with the same V-cycle as RIGHT preconditioner — the alternative outer solver the paper names as
// future work (section 6).  Notation of the textbook algorithm (Saad, Iterative Methods, Alg. 7.7, preconditioned
// on the right: y = M p, z = M s):
//     r0 = b - A x0, rhat = r0, rho = alpha = omega = 1, v = p = 0
//     rho' = (rhat, r); beta = (rho'/rho)(alpha/omega); p = r + beta (p - omega v)
//     y = M p; v = A y; alpha = rho' / (rhat, v); s = r - alpha v            [|s|/|b| < rtol: x += alpha y, stop]
//     z = M s; t = A z; omega = (t, s)/(t, t); x += alpha y + omega z; r = s - omega t     [|r|/|b| < rtol: stop]
// Stop test and restarts follow rules K1, K3, K5 of the fGMRES solve: Eq. 23 on the recurrence residual inside,
// the recomputed true residual decides at the end; if it is still >= rtol the iteration restarts from it (rhat = r = b - A x).
// iters counts preconditioner applications (two per full step), as orc_solve_ex does.  precond as there (0 cycle, 1 identity,
// 2 dense exact inverse).  hist[k] = recurrence |s| or |r| over |b| after application k+1.
// Returns 0 converged, 1 max_iters reached, 2 breakdown (rho, (rhat, v) or (t, t) vanished), <0 error.
int orc_solve_bicgstab(void* h, const double* f_user, const double* x0_user, double* x_user, double rtol, int precond,
                       int* iters_out, double* relres_out, double* hist) {
    Oracle* o = (Oracle*)h;
    if (!o->have_coeffs) { g_err = "solve before update"; return -3; }
    Level& lv = o->lev[0];
    const int64_t n = lv.n;
    std::vector<double> b(n), x(n), r(n), rhat(n), p(n, 0.0), v(n, 0.0), y(n), s(n), z(n), t(n);
    for (int64_t k = 0; k < n; k++) { b[o->user2canon[k]] = f_user[k]; x[o->user2canon[k]] = x0_user[k]; }
    if (precond == 2 && o->lu0.empty()) { assemble_dense(lv, o->lu0); if (!lu_factor(o->lu0, o->piv0, n)) return -2; }
    auto M = [&](const std::vector<double>& in, std::vector<double>& out) {
        if (precond == 0) { std::fill(out.begin(), out.end(), 0.0); mg_cycle(*o, 0, out.data(), in.data(), o->gamma); }
        else if (precond == 1) out = in;
        else lu_solve(o->lu0, o->piv0, n, in.data(), out.data());
    };
    int iters = 0, status = 1; double relres = 0.0;
    const double bn = std::sqrt(dot(b.data(), b.data(), n));
    auto finish = [&](int st) {
        for (int64_t k = 0; k < n; k++) x_user[k] = x[o->user2canon[k]];
        if (iters_out) *iters_out = iters;
        if (relres_out) *relres_out = relres;
        return st;
    };
    if (bn == 0.0) { std::fill(x.begin(), x.end(), 0.0); return finish(0); }                     // K1
    while (true) {
        apply(lv, x.data(), r.data());
        for (int64_t k = 0; k < n; k++) r[k] = b[k] - r[k];                                      // D4
        relres = std::sqrt(dot(r.data(), r.data(), n)) / bn;
        if (relres < rtol) { status = 0; break; }                                                // K1 / K5
        if (iters >= o->max_iters) { status = 1; break; }
        rhat = r;
        std::fill(p.begin(), p.end(), 0.0); std::fill(v.begin(), v.end(), 0.0);
        double rho = 1.0, alpha = 1.0, omega = 1.0;
        bool breakdown = false;
        while (iters < o->max_iters) {
            const double rho1 = dot(rhat.data(), r.data(), n);
            if (rho1 == 0.0 || omega == 0.0) { breakdown = true; break; }
            const double beta = (rho1 / rho) * (alpha / omega);
            for (int64_t k = 0; k < n; k++) p[k] = r[k] + beta * (p[k] - omega * v[k]);
            M(p, y);
            apply(lv, y.data(), v.data());
            const double rv = dot(rhat.data(), v.data(), n);
            if (rv == 0.0) { breakdown = true; break; }
            alpha = rho1 / rv;
            for (int64_t k = 0; k < n; k++) s[k] = r[k] - alpha * v[k];
            iters++;
            const double sn = std::sqrt(dot(s.data(), s.data(), n)) / bn;
            if (hist) hist[iters - 1] = sn;
            if (sn < rtol || iters >= o->max_iters) {                                             // K3 at the half step
                for (int64_t k = 0; k < n; k++) x[k] += alpha * y[k];
                break;
            }
            M(s, z);
            apply(lv, z.data(), t.data());
            const double tt = dot(t.data(), t.data(), n);
            if (tt == 0.0) { for (int64_t k = 0; k < n; k++) x[k] += alpha * y[k]; breakdown = true; break; }
            omega = dot(t.data(), s.data(), n) / tt;
            for (int64_t k = 0; k < n; k++) { x[k] += alpha * y[k] + omega * z[k]; r[k] = s[k] - omega * t[k]; }
            iters++;
            rho = rho1;
            const double rn = std::sqrt(dot(r.data(), r.data(), n)) / bn;
            if (hist) hist[iters - 1] = rn;
            if (rn < rtol) break;                                                                 // K3
        }
        if (breakdown) {
            apply(lv, x.data(), r.data());
            for (int64_t k = 0; k < n; k++) r[k] = b[k] - r[k];
            relres = std::sqrt(dot(r.data(), r.data(), n)) / bn;
            status = relres < rtol ? 0 : 2;
            break;
        }
    }                                                                                             // K5: loop = restart
    return finish(status);
}

}  // extern "C"
