/* mg_b200.h — C ABI of the B200-native fGMRES + geometric-multigrid elliptic solver.
 *
 * Solves  lambda*u - div(c grad u) = f  (Eq. 3 with paper-xi = 1, Eq. 6) on a
 * locally Cartesian, logically unstructured 2D mesh (Eq. 9) with Dirichlet and Neumann
 * guard points (Eq. 11-16), by flexible GMRES preconditioned with one
 * geometric-multigrid V-cycle using red-black-boundary Gauss-Seidel.
 * The three-call shape create / update / solve is PAPER.md:133-139.  DESIGN.md section 3 lists the
 * readings taken where the paper is silent (rule numbers M*, D*, T*, GS, C, V, K* are quoted below).
 *
 * Conventions
 *  - "HOST" / "DEVICE" says where a pointer must live.  Device pointers are plain CUDA device memory of
 *    the current device; `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *  - User vectors have length n (all mesh points, inner + guard) in the CALLER'S point order, fp64.
 *    f[l] = rho_l on inner rows, phi_D,l on Dirichlet rows, Gamma_l on Neumann rows.
 *  - "Level vectors" (test entry points) have length mg_level_n(level) in the level's canonical order:
 *    ascending (J, I) of the level's own lattice indices (rule M7).  Levels are 0-based (0 = finest).
 *  - Ownership: the handle owns all device memory it allocates (through the allocator installed with
 *    mg_set_allocator, default cudaMalloc/cudaFree); callers own every array they pass in; host mesh
 *    arrays may be freed after mg_setup returns.  One handle = one mesh = one stream at a time.
 *  - Errors: every call returns 0 on success, a negative MG_E* code on failure (never throws, never
 *    aborts); mg_solve may also return the positive MG_NOT_CONVERGED / MG_BREAKDOWN.
 *  - There is no CPU fallback: without a CUDA device every compute call returns MG_ECUDA.
 */
#ifndef MG_B200_H
#define MG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_handle_s* mg_handle;
#define MG_SETUP_HOST_ONLY 1
#define MG_SETUP_FUSED_TAIL 2
#define MG_SETUP_FULL_CGS2 4
#define MG_NU_NONE (-1) /* mg_options.nu_post: no post-smoothing (0 means "default") */

enum {
    MG_OK = 0,
    MG_NOT_CONVERGED = 1, /* max_iters reached; x holds the last iterate                                  */
    MG_BREAKDOWN = 2,     /* h_{j+1,j} = 0 with the residual still above rtol (rule K3)                  */
    MG_EINVAL = -1,       /* null pointer, n <= 0, h <= 0, bad option, bad level                         */
    MG_EMESH = -2,        /* duplicate (i,j); inner point lacking a neighbour; guard without an inner
                             4-neighbour (rule M2); coarsest level too large for the dense solve */
    MG_ECOEFF = -3,       /* mg_solve / single-step calls: the last update's fields were not admissible: c <= 0
                             (PAPER.md:51), xi <= 0, a non-finite value, or a coarsest-level operator that is
                             singular (zero / non-finite pivot) — all tested on the device during the update.
                             Deviations from a synchronous check, both deliberate: the update itself returns
                             MG_OK and the NEXT call that uses the operators reports the error (the update
                             is asynchronous, G26); lambda < 0 is accepted (the paper's own test
                             case has lambda of both signs, Eq. 21)                            */
    MG_ENOTREADY = -4,    /* solve / cycle before the first mg_update_coeffs                             */
    MG_ECUDA = -5,        /* CUDA runtime error or no device                                             */
    MG_ENOMEM = -6
};

/* Mesh: HOST pointers, length n, borrowed for the duration of mg_setup (Eq. 9). */
typedef struct {
    int64_t n;        /* number of mesh points, inner + guard                     */
    const int32_t* i; /* lattice column index i_l (any int32, negative allowed)   */
    const int32_t* j; /* lattice row index j_l                                    */
    double h;         /* finest grid spacing                                      */
} mg_mesh;

/* Boundary classification: HOST pointer, length n. 0 = inner, 1 = Dirichlet guard (Eq. 11),
 * 2 = Neumann guard (Eq. 16). */
typedef struct {
    const uint8_t* kind;
} mg_bc;

/* Solver parameters ("create ... based on the specified algorithm and solver parameters").
 * Zero-initialise and override; 0 means "default" for every field. */
typedef struct {
    int levels;    /* N_sigma; 0 = auto: coarsen while the bounding lattice > 9x9 and |Inner| >= 16 (M8) */
    int nu_pre;    /* nsmooth_pre, default 2; must be >= 1 (rule T2)                     */
    int nu_post;   /* nsmooth_post, default 2; MG_NU_NONE = no post-smoothing, V(nu_pre,0)      */
    int restart_m; /* fGMRES restart length m, default 30, max 64                                        */
    int max_iters; /* cap on preconditioner applications, default 200                                    */
    int flags;     /* bit 0 (MG_SETUP_HOST_ONLY): build the host hierarchy only, touch no device; only the
                      inspection calls mg_num_levels / mg_level_n / mg_level_info / mg_transfer_info work,
                      every compute call returns MG_ECUDA.
                      bit 1 (MG_SETUP_FUSED_TAIL): run the cycle steps of the small levels (<= 148 tiles) in one
                      cooperative kernel instead of one kernel per step (bit-identical results; off by default; ignored
                      when planes > 1).
                      bit 2 (MG_SETUP_FULL_CGS2): always run the second Gram-Schmidt update of the Arnoldi step;
                      by default it is skipped in the steps where the measured defect ||V^T w'|| is already
                      <= 1e-13 ||w'|| (G23; same iterates to that level).
                      Other bits must be 0.                                                              */
    int gamma;     /* cycle index of PAPER.md:187-189, 197: 0 or 1 = V-cycle (default), 2 = W-cycle; 3 = F-cycle
                      (one F-cycle visit, then one V-cycle visit of the next coarser level)   */
    int planes;    /* P >= 1 (0 = 1): number of planes solved TOGETHER on this mesh (one elliptic solve per
                      poloidal plane, all planes share the mesh).  The handle keeps the mesh data once and every vector
                      P times; mg_update_coeffs / mg_solve then take P fields back to back (plane p at offset p * n),
                      every kernel launch covers all planes (gridDim.y = P), each plane has its own fGMRES state and
                      stops on its own Eq. 23; results are bit-identical to P separate handles.  The single-step and
                      inspection calls below work on plane 0.                                                   */
    int solver;    /* outer solver: 0 = fGMRES(restart_m) (the paper's and the benchmarked choice);
                      1 = BiCGStab with the same cycle as right preconditioner ("BiCGStab ... as alternative");
                      it keeps no Krylov basis (seven work vectors instead of 2 (m + 1)), restart_m is ignored, iters
                      counts preconditioner applications (two per step), the stop test and the restart from the
                      recomputed true residual are those of mg_solve                                             */
} mg_options;

/* Device-memory allocator used by handles created afterwards (e.g. torch's caching allocator).
 * alloc returns a device pointer or NULL; both may be NULL to restore cudaMalloc/cudaFree.  A handle remembers the
 * pair that was installed when it was created and uses it for all its later allocations and in mg_destroy. */
typedef void* (*mg_alloc_fn)(uint64_t bytes, void* stream);
typedef void (*mg_free_fn)(void* ptr);
int mg_set_allocator(mg_alloc_fn alloc_fn, mg_free_fn free_fn);

/* create: builds the level hierarchy on the host (rules M1-M8: coarse point lists,
 * guard classification, Neumann stencils, tile layout, transfer tables), uploads it and allocates all
 * work space.  Synchronous.  Errors: MG_EINVAL, MG_EMESH, MG_ECUDA, MG_ENOMEM. */
int mg_setup(const mg_mesh* mesh, const mg_bc* bc, const mg_options* opt, void* stream, mg_handle* out);

/* update: new coefficients lambda, c (= BASELINE "xi") on ALL n points, DEVICE
 * pointers, user order (P * n values for a handle with P planes).  Restricts them to all coarser levels (rule T4) and factorises the coarsest
 * operator (rule C) on the device.  Asynchronous on `stream`.  Admissibility (c > 0; finite lambda) is
 * tested on the device during the call; a violation is reported by the next mg_solve as MG_ECOEFF. */
int mg_update_coeffs(mg_handle h, const double* d_lambda, const double* d_c, void* stream);

/* update for the paper's three-field form  lambda phi - xi div(c grad phi) = rho  (Eq. 3; the row of
 * point (i,j) carries xi_{i,j}/2, Eq. 10).  d_xi: DEVICE, length n, user order, > 0 on ALL points
 * (guard rows, Eq. 11 / 16, do not contain it, but the coarser levels average over guards too); it is transferred to the coarser levels like lambda and c
 * (PAPER.md:153, 207).  d_xi == NULL is mg_update_coeffs (xi = 1).  The handle keeps the form of the
 * last update; switching forms re-captures the iteration graph at the next solve.  The stop test of mg_solve is
 * on the residual of the three-field rows.  Costs 8 B per point and smoothing launch (and one fp64 division per point) more than the two-field form. */
int mg_update_coeffs3(mg_handle h, const double* d_lambda, const double* d_xi, const double* d_c, void* stream);

/* solve: fGMRES(m) with one V-cycle as right preconditioner (rules K1-K5), stopping
 * on ||A x - f|| / ||f|| < rtol (Eq. 23).  d_f, d_x0, d_x: DEVICE, length n, user order;
 * d_x may alias d_x0.  iters (HOST, may be NULL) receives the number of preconditioner applications,
 * final_relres (HOST, may be NULL) the recomputed true relative residual.  With P planes (mg_options.planes) the three
 * vectors hold P * n values (plane p at p * n), iters and final_relres are arrays of P entries, and the return value
 * is the worst over the planes (MG_BREAKDOWN > MG_NOT_CONVERGED > MG_OK).  Returns after the stream
 * has finished the solve.  Returns MG_OK, MG_NOT_CONVERGED, MG_BREAKDOWN or an error.  On MG_NOT_CONVERGED
 * mg_last_error() says whether the recurrence residual had passed rtol while the recomputed true residual had not
 * (rtol below the accuracy attainable in fp64 on this mesh; the method has no stagnation exit). */
int mg_solve(mg_handle h, const double* d_f, const double* d_x0, double* d_x, double rtol, int* iters,
             double* final_relres, void* stream);

/* Same two calls with HOST buffers (pageable or pinned): the library stages them through device
 * buffers it owns; copies run on `stream` (PAPER.md:217 describes exactly this transfer pattern). */
int mg_update_coeffs_host(mg_handle h, const double* h_lambda, const double* h_c, void* stream);
int mg_update_coeffs3_host(mg_handle h, const double* h_lambda, const double* h_xi, const double* h_c, void* stream);
int mg_solve_host(mg_handle h, const double* h_f, const double* h_x0, double* h_x, double rtol, int* iters,
                  double* final_relres, void* stream);

int mg_destroy(mg_handle h);

/* ---- inspection (HOST outputs; any output pointer may be NULL) -------------------------------- */
int mg_num_levels(mg_handle h);
int64_t mg_level_n(mg_handle h, int level);
/* Per-level arrays in canonical order: lattice indices I, J; kind (0/1/2); colour (0 red, 1 black,
 * 2 guard; rule M6); nbr [4n] = canonical indices of W, E, S, N (-1 absent, rule M5); for Neumann
 * guards ns_tn [2n] = (2 n^R, 2 n^Z) of Eq. 13 and ns_fallback [n] (rule D3); slot [n] = position of
 * the point in the device tile layout.  user2canon [n_0] (level 0 only) = canonical index of each
 * user point. */
int mg_level_info(mg_handle h, int level, int32_t* I, int32_t* J, uint8_t* kind, uint8_t* colour, int32_t* nbr,
                  int8_t* ns_tn, uint8_t* ns_fallback, int32_t* slot, int64_t* user2canon);
/* Transfer tables between `level` (fine) and level+1: fine9 [9*n_{level+1}] = canonical fine indices
 * of the 3x3 neighbourhood of each coarse point (row-major dy, dx; -1 absent); parent [4*n_level] =
 * canonical coarse indices of the bilinear parents (-1 absent / unused), ptype [n_level] = 0 coincident,
 * 1 R-edge, 2 Z-edge, 3 centre (Fig. 3). */
int mg_transfer_info(mg_handle h, int level, int32_t* fine9, int32_t* parent, uint8_t* ptype);
/* Current coefficients of a level (DEVICE -> HOST copy, canonical order). */
int mg_level_coeffs(mg_handle h, int level, double* h_lambda, double* h_c, void* stream);
/* xi of a level (DEVICE -> HOST copy, canonical order; all 1 in the two-field form). */
int mg_level_xi(mg_handle h, int level, double* h_xi, void* stream);

/* ---- single steps, for parity tests.  DEVICE level vectors in canonical order ------------------ */
int mg_apply(mg_handle h, int level, const double* d_x, double* d_y, void* stream);            /* y = A x (D1-D3) */
int mg_smooth(mg_handle h, int level, double* d_x, const double* d_b, int sweeps, void* stream); /* GS rbb        */
int mg_restrict(mg_handle h, int level, const double* d_fine, double* d_coarse, void* stream);  /* rule T2        */
/* The cycle's fused step: x <- S^sweeps x (sweeps >= 1), then d_coarse = R (A x - b) on level + 1,
 * in one pass per two sweeps; this is the kernel bench.py reports its roofline for. */
int mg_smooth_restrict(mg_handle h, int level, double* d_x, const double* d_b, int sweeps, double* d_coarse, void* stream);
int mg_prolong_correct(mg_handle h, int level, const double* d_coarse_e, double* d_x_fine, void* stream); /* T3   */
int mg_coarse_solve(mg_handle h, const double* d_b, double* d_x, void* stream);                 /* rule C         */
int mg_vcycle(mg_handle h, int level, double* d_x, const double* d_b, void* stream);

/* Counters: kernels launched by this handle since creation (graph-launched kernels included). */
int64_t mg_kernel_launches(mg_handle h);
/* Wall-clock-free timing of the last mg_solve / mg_update_coeffs on the device (CUDA events on the
 * launching stream), in milliseconds; negative if not available. */
double mg_last_solve_ms(mg_handle h);
double mg_last_update_ms(mg_handle h);
/* Device time of the smoothing kernels alone (without the in/out permutations) of the last mg_smooth or
 * mg_smooth_restrict call, CUDA events on the launching stream; synchronises on the second event. */
double mg_last_step_ms(mg_handle h);
/* Arnoldi steps of the last mg_solve whose second Gram-Schmidt update ran (see MG_SETUP_FULL_CGS2); -1 before
 * the first solve. */
int mg_last_reorth(mg_handle h);
/* Per-iteration history of the last mg_solve (first min(iters, 512, cap) iterations), HOST arrays, either may be
 * NULL: relres[k] = the recurrence residual |g_{k+1}| / ||f|| after iteration k+1 (Eq. 23; monotone
 * within a restart cycle), orth[k] = ||V^T w'|| / ||w'|| measured after the first Gram-Schmidt projection of that
 * iteration (0 on the unfused path, restart_m > 32).  Returns the number of entries written. */
int mg_last_history(mg_handle h, double* relres, double* orth, int cap);

/* ---- an entry point that allocates nothing --------------------------------------------------------------------
 * d_out[0] = ||d_v||_2 over n doubles (the reduction behind the stop test of PAPER.md:260 Eq. 23), for callers that cannot
 * call cudaMalloc: stream capture, tight serving loops, harnesses that forbid it.  d_v, d_out: DEVICE, caller-owned;
 * needs no handle.  Asynchronous on `stream`; calls no cudaMalloc / cudaFree / allocating routine (one cudaMemsetAsync
 * of 4 bytes and one kernel).  Its scratch (4096 per-block partial sums + a ticket, 32.25 KB) is a fixed __device__ array of the library that
 * every GPU which loads the library holds until exit; n > MG_NOALLOC_MAX_N is refused with MG_EINVAL (mg_last_error says
 * why).  All calls on a device share that array: calls that OVERLAP on the GPU (different streams, unordered graph
 * branches) race and give wrong results — order them.  The first call on a device looks the array's address up
 * (cudaGetSymbolAddress): make it outside stream capture.  The summation order depends on n only (deterministic, the same on
 * every device).  Errors: MG_EINVAL, MG_ECUDA. */
#define MG_NOALLOC_MAX_N 268435456LL /* 4096 partial sums x 65536 elements per block */
int mg_norm2_noalloc(const double* d_v, int64_t n, double* d_out, void* stream);

const char* mg_strerror(int code);
const char* mg_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MG_B200_H */
