// Device-side structures and kernel launch wrappers of libmg_b200 (internal).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "mg_common.h"

namespace mgb {

constexpr int MAX_M = 64;          // largest fGMRES restart length
constexpr int RED_BLOCKS_MAX = 1024;   // capacity of the per-block partial sums of the grid-wide reductions
constexpr int RED_THREADS = 256;

// text behind mg_last_error() of the calling thread (mg_api.cu), for entry points that live in other files
void set_last_error(const std::string& msg);

// Per-device facts, queried once per device (mg_devinfo.cu).
struct DevInfo {
    int device;
    int sms;     // cudaDevAttrMultiProcessorCount (148 on B200)
    int coop;    // cooperative launch supported
};
const DevInfo& dev_info();                                       // of the calling thread's current device
cudaError_t ensure_dyn_smem(const void* func, size_t bytes);     // opt-in dynamic shared memory, once per (kernel, device)
inline int red_blocks() { const int b = 4 * dev_info().sms; return b < RED_BLOCKS_MAX ? b : RED_BLOCKS_MAX; }   // blocks of the grid-wide reductions

// One multigrid level on the device (all pointers device memory; vectors have nslots entries).
struct LevelDev {
    int32_t ntiles;
    int32_t ntiles_fine;     // null-tile id of the next finer level (for ctab), 0 on level 0
    int32_t ntiles_coarse;   // null-tile id of the next coarser level (for ptab)
    int64_t nslots;
    double h, kappa;         // kappa = 1 / (2 h^2), rule D1
    const uint16_t* code;
    const int32_t* tnb;      // 9 per tile
    const int32_t* ctab;     // 9 per tile (this level as the coarse side)
    const int32_t* ptab;     // 9 per tile (this level as the fine side): coarse tiles around the parent tile
    const int32_t* tij;      // 2 per tile: tile coordinates (TI, TJ)
    const uint8_t* tflag;    // per tile: bits 0 / 1 / 2 = every cell within 2 / 4 / 6 cells of the tile is an inner point
    const int32_t* tlist[2]; // tile ids, [nint[k] interior | ngen[k] general | overflow tiles], by flag bit 1 (k = 0) / bit 2 (k = 1)
    int32_t nint[2], ngen[2];
    const int32_t* smeta[2]; // per interior and general tile of tlist[k], in list order: 24 ints {tnb[9], ptab[9], TI & 1, TJ & 1, tile id, pad} (mg_strip_gs.cuh)
    double* lam;
    double* c;
    double* rd;              // 1 / a_ll on inner points (rule D1), 0 elsewhere; derived at every update (U2)
    // Three-field form lambda phi - xi div(c grad phi) = rho (Eq. 3; Eq. 10 PAPER.md:82 carries xi_{i,j}/2
    // of the row's own point).  Null in the two-field form (xi = 1).  With xi the smoother works on
    // the row divided by xi: it holds b / xi in registers and rd holds xi / a_ll, so its sweeps are unchanged.
    double* xi;              // xi on every present point (grid-transferred like lambda and c)
};

// fGMRES state, resident on the device (rules K1-K5).  Givens rotations, the least-squares
// right-hand side and the stop test live here so that no iteration needs the host.
struct GmresState {
    int j;            // current column (0-based) of the running restart cycle
    int iters;        // preconditioner applications so far
    int status;       // 0 running, 1 converged, 2 max_iters, 3 breakdown
    int cycle_end;    // 1: the running cycle ended (converged, j == m, max_iters or breakdown)
    int m, max_iters;
    int ticket;       // last-block-done counter of the grid reductions
    int nreorth;      // Arnoldi steps of this solve whose second Gram-Schmidt update ran
    int skip2;        // 1: the step in flight needs no second update (k_final_v only normalises)
    int pad;
    double reorth_tol;  // second update skipped when ||V^T w'|| <= reorth_tol ||w'||; < 0: never (MG_SETUP_FULL_CGS2)
    double rtol, bn, beta, relres, hn, inv_hn;
    double red[MAX_M + 2];          // results of the last multi-reduction
    double hcol[MAX_M + 2];         // Hessenberg column being built (h_0j .. h_j+1,j)
    double H[(MAX_M + 1) * MAX_M];  // rotated Hessenberg (upper triangular R), row-major, ld = MAX_M
    double g[MAX_M + 1], cs[MAX_M], sn[MAX_M], y[MAX_M];
    double hist[512];               // |g_{k+1}| / bn per iteration
    double orth[512];               // ||V^T w'|| / ||w'|| after the first Gram-Schmidt projection, per iteration (fused path)
    // BiCGStab (mg_options.solver = 1, mg_bicgstab.cu): the scalars of the recurrence and the flags of the running step
    double b_rho, b_rho1, b_alpha, b_omega;
    int b_first;                    // first step after a (re)start: p = r
    int b_half;                     // the step ends after its first half (|s| below rtol, iteration cap, or (t, t) = 0)
    int b_skip2;                    // second preconditioner application of the step not needed (b_half or cycle_end)
    int b_pad;
};

// Planes (one elliptic solve per poloidal plane, all on the same mesh).  A handle created
// with P planes keeps the mesh data (codes, tile tables) once and every vector P times, plane p at p * (plane stride);
// all kernels take the plane from blockIdx.y, so one launch (one captured graph) serves all planes, each with its own
// fGMRES state and convergence flag.
constexpr int ST_INTS = (int)(sizeof(GmresState) / sizeof(int));   // distance between the states of two planes, in ints

// A vector that may be one column of a Krylov basis selected on the device:
// address = base + plane * pstride + (idx ? idx[plane * ST_INTS] + off : 0) * stride.
struct VecRef {
    double* base;
    int64_t stride;
    const int* idx;
    int off;
    int64_t pstride;
};
__host__ __device__ inline VecRef vec(double* p, int64_t pstride = 0) { return VecRef{p, 0, nullptr, 0, pstride}; }
#ifdef __CUDACC__
__device__ __forceinline__ double* resolve(const VecRef& v, int plane = 0) {
    return v.base + plane * v.pstride + (v.idx ? (int64_t)(v.idx[(int64_t)plane * ST_INTS] + v.off) * v.stride : 0);
}
// plane p of a level: the coefficient arrays advance by p * nslots; codes and tile tables are shared
__device__ __forceinline__ LevelDev plane_of(LevelDev lv, int p) {
    const int64_t o = (int64_t)p * lv.nslots;
    lv.lam += o; lv.c += o; lv.rd += o;
    if (lv.xi) lv.xi += o;
    return lv;
}
// Inner row of rule D1 in difference form, lambda x_l + a_W (x_l - x_W) + a_E (x_l - x_E) + a_S (x_l - x_S) + a_N (x_l - x_N),
// with the rounding sequence spelled out (one product, four fused multiply-adds in the order W, E, S, N) so that every
// kernel that evaluates a row — stand-alone, fused into a smoother launch, shared-memory or register-tiled — produces the
// same bits and the choice of kernel (level size, number of planes) never shows in a result.
__device__ __forceinline__ double row_d1(double lam, double xl, double aW, double xW, double aE, double xE, double aS, double xS,
                                         double aN, double xN) {
    double r = __dmul_rn(lam, xl);
    r = __fma_rn(aW, __dsub_rn(xl, xW), r);
    r = __fma_rn(aE, __dsub_rn(xl, xE), r);
    r = __fma_rn(aS, __dsub_rn(xl, xS), r);
    r = __fma_rn(aN, __dsub_rn(xl, xN), r);
    return r;
}
// Eq. 16 solved for the guard point, x_l = (sum_{k != l} w_k x_k - delta b_l) / (1 - w_l), rounding sequence fixed likewise
__device__ __forceinline__ double neumann_point(double sum, double delta, double b, double wself) {
    return __ddiv_rn(__fma_rn(-delta, b, sum), __dsub_rn(1.0, wself));
}
__device__ __forceinline__ bool stopped(const int* stop, int plane) { return stop != nullptr && stop[(int64_t)plane * ST_INTS] != 0; }
#endif

struct Launch {
    cudaStream_t stream;
    int64_t* counter;   // host counter of kernel launches (may be null)
    const int* stop = nullptr;   // device flag of plane 0 (plane p: stop[p * ST_INTS]): V-cycle kernels return at once when it is
                                 // set (iterations enqueued ahead of the convergence test), null = always run
    int planes = 1;              // gridDim.y of every launch
};

// ---- tile kernels (mg_kernels.cu) ----
// mode 0: y = A x      1: y = b - A x      2: y = A x - b
void launch_apply(const Launch& L, const LevelDev& lv, VecRef x, VecRef b, VecRef y, int mode);
// `sweeps` (1 or 2) full red-black-boundary Gauss-Seidel sweeps in ONE pass over memory: x_out = S^sweeps x_in.
// x_in and x_out must be different buffers (halo cells are recomputed by neighbouring CTAs);
// x_in_zero: treat x_in as the zero vector without reading it.
// coarse != null: the launch also writes d_coarse = R (A x_out - b) on that level, fused.
void launch_gs_fused(const Launch& L, const LevelDev& lv, VecRef x_in, VecRef x_out, VecRef b, int sweeps, bool x_in_zero,
                     const LevelDev* coarse = nullptr, double* d_coarse = nullptr, double* w_out = nullptr);
// Same, preceded in the same pass by the coarse-grid correction x_in - P e_c with set_bnds_hom (rule T3).
// w_out != null (either call): the launch also writes w_out = A x_out (the Arnoldi step's operator apply, fused).
void launch_gs_correct(const Launch& L, const LevelDev& lv, const double* e_coarse, VecRef x_in, VecRef x_out, VecRef b, int sweeps,
                       double* w_out = nullptr);
void launch_copy(const Launch& L, VecRef src, VecRef dst, int64_t n);
void launch_restrict(const Launch& L, const LevelDev& fine, const LevelDev& coarse, const double* d_fine, double* d_coarse);
// d_coarse = R (A x - b), the defect never stored (rules D4 + T2)
void launch_defect_restrict(const Launch& L, const LevelDev& fine, const LevelDev& coarse, VecRef x, VecRef b, double* d_coarse);
void launch_prolong_correct(const Launch& L, const LevelDev& fine, const LevelDev& coarse, const double* e_coarse,
                            double* e_fine_tmp, VecRef x_fine);
void launch_restrict_coeff(const Launch& L, const LevelDev& fine, const LevelDev& coarse);
void launch_diag(const Launch& L, const LevelDev& lv);   // U2: rd = 1 / a_ll from lambda, c
void launch_zero(const Launch& L, VecRef x, int64_t n);
// ps: distance between the planes of the tiled vector (user vectors: n)
void launch_gather(const Launch& L, const double* src, const int32_t* slot, double* dst_tiled, int64_t n, int64_t ps);   // dst[slot[k]] = src[k]
void launch_gather_check(const Launch& L, const double* src, const int32_t* slot, double* dst_tiled, int64_t n, int64_t ps, int mode, int bit, int* bad);
void launch_scatter(const Launch& L, const double* src_tiled, const int32_t* slot, double* dst, int64_t n, int64_t ps);  // dst[k] = src[slot[k]]

// ---- fused small levels (mg_tail.cu): the cycle steps of all levels >= s0 as a program run by one
// cooperative kernel, grid.sync() between steps
// per (level, tile) tables a CTA of the fused kernel preloads once: ints
//   [META_TN..+9) neighbour tiles, [META_PT..+9) coarse parent tiles, [META_ODD..+2) tile parity, [META_FLAG] interior flags,
//   this tile as the COARSE side of a defect restriction: [META_CT..+9) fine tiles, [META_FTN..+36) neighbour tables
//   of the 2 x 2 fine tiles, [META_RING..+20) W,E,S,N neighbours of the SW, W, W', S, S' ring tiles
enum { META_TN = 0, META_PT = 9, META_ODD = 18, META_FLAG = 20, META_CT = 21, META_FTN = 30, META_RING = 66, META_INTS = 88 };
constexpr int TAIL_MAX_LEVELS = 16;
enum { TAIL_GS = 0, TAIL_DR = 1, TAIL_COARSE = 2, TAIL_COPY = 3 };
#define TAIL_TOPX (reinterpret_cast<double*>(1))   // placeholder: the cycle's x vector (a VecRef resolved on the device)
#define TAIL_TOPB (reinterpret_cast<double*>(2))   // placeholder: the cycle's right-hand side
struct TailOp {
    unsigned char type, level, ns, pc;   // level: the (fine) level the step works on; pc: 1 correction first, 2 defect restriction after
    int zero;                            // GS: x_in is the zero vector
    int ntiles;                          // tiles the step loops over
    double *a, *b, *c;                   // GS: x_in, x_out, rhs; DR: x, coarse defect out, rhs; COARSE: rhs, x; COPY: src, dst
    const double* ec;                    // GS with correction: coarse-level solution
    double* dc;                          // GS with fused defect restriction (pc = 2): restricted defect on level + 1
    int64_t n;                           // COPY: length
};
constexpr int TAIL_MAX_OPS = 48;
struct TailProgram {
    int nops;
    TailOp op[TAIL_MAX_OPS];
};
struct TailCoarse {
    const double* Ainv;
    const int32_t* cslot;
    int n;
};
int tail_max_grid();   // largest co-resident grid of the fused kernel (0: cooperative launch unavailable)
// levels s0 .. nlev-1 take part; grid must be >= the tile count of every step (one tile per CTA)
cudaError_t launch_tail(const Launch& L, const LevelDev* d_levs, int s0, int nlev, const TailProgram& prog, const TailCoarse& cs,
                        VecRef topx, VecRef topb, int grid);

// ---- coarsest level (mg_coarse.cu) ----
// doubles of work space per plane: [A | I] (n x 2n) + the published pivot column (x 2) + pivots
__host__ __device__ inline size_t coarse_work_doubles(int n) { return 2 * (size_t)n * n + 2 * (size_t)n + 2; }
void launch_coarse_factor(const Launch& L, const LevelDev& lv, const int32_t* cslot, const int32_t* slot2row, int n,
                          double* work /* n x 2n */, double* Ainv /* n x n */, int* bad /* bit 3 set on a zero / non-finite pivot */);
void launch_coarse_solve(const Launch& L, const double* Ainv, const int32_t* cslot, int n, VecRef b_tiled, VecRef x_tiled);

// ---- fGMRES vector kernels (mg_krylov.cu) ----
void launch_norm2(const Launch& L, const double* v, int64_t n, GmresState* st, double* partial, int which);  // which: 0 -> bn, 1 -> beta
void launch_start_cycle(const Launch& L, GmresState* st, const double* r, double* V0, int64_t n);
void launch_multidot(const Launch& L, const double* w, const double* V, int64_t stride, int64_t n, GmresState* st, double* partial, int m);
void launch_update_w(const Launch& L, double* w, const double* V, int64_t stride, int64_t n, GmresState* st, double* partial, int pass);
void launch_givens(const Launch& L, GmresState* st);
// fused CGS2 for restart lengths m <= MAX_M_FUSED (three passes over the basis, Givens inside the second)
constexpr int MAX_M_FUSED = 32;
void launch_update_dot(const Launch& L, double* w, const double* V, int64_t stride, int64_t n, GmresState* st, double* partial);
void launch_final_v(const Launch& L, const double* w, double* V, int64_t stride, int64_t n, GmresState* st);
void launch_next_v(const Launch& L, const double* w, double* V, int64_t stride, int64_t n, GmresState* st);
void launch_update_x(const Launch& L, double* x, const double* Z, int64_t stride, int64_t n, GmresState* st);
void launch_zero_rhs_planes(const Launch& L, double* x, int64_t n, const GmresState* st);
// ---- BiCGStab vector kernels (mg_bicgstab.cu); all vectors level-0 tile layout, n = nslots, plane stride n
void launch_bi_start(const Launch& L, GmresState* st, const double* r, double* rhat, int64_t n);
void launch_bi_p(const Launch& L, GmresState* st, const double* r, double* p, const double* v, int64_t n);
void launch_bi_alpha(const Launch& L, GmresState* st, const double* rhat, const double* v, int64_t n, double* partial);
void launch_bi_s(const Launch& L, GmresState* st, const double* r, const double* v, double* s, int64_t n, double* partial);
void launch_bi_omega(const Launch& L, GmresState* st, const double* t, const double* s, int64_t n, double* partial);
void launch_bi_update(const Launch& L, GmresState* st, double* x, double* r, const double* rhat, const double* y, const double* z,
                      const double* s, const double* t, int64_t n, double* partial);
void launch_init_state(const Launch& L, GmresState* st, int m, int max_iters, double rtol, bool full_cgs2);

}  // namespace mgb
