// C-ABI layer of libmg_b200 (include/mg_b200.h): handle, device hierarchy upload, V-cycle and fGMRES
// orchestration (CUDA graph per Arnoldi iteration), inspection and single-step test entry points.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mg_b200.h"
#include "mg_device.h"

using namespace mgb;

namespace {

thread_local std::string g_last_error;
mg_alloc_fn g_alloc = nullptr;
mg_free_fn g_free = nullptr;

#define CU(call)                                                                             \
    do {                                                                                     \
        cudaError_t e__ = (call);                                                            \
        if (e__ != cudaSuccess) {                                                            \
            g_last_error = std::string(#call) + ": " + cudaGetErrorString(e__);              \
            return MG_ECUDA;                                                                 \
        }                                                                                    \
    } while (0)

struct LevelBuf {           // device arrays owned per level
    uint16_t* code = nullptr;
    uint8_t* tflag = nullptr;
    int32_t *tnb = nullptr, *ctab = nullptr, *ptab = nullptr, *tij = nullptr, *canon2slot = nullptr, *tlist[2] = {nullptr, nullptr}, *smeta[2] = {nullptr, nullptr};
    double* xi = nullptr;   // three-field form only: allocated by the first mg_update_coeffs3 with xi
    double *lam = nullptr, *c = nullptr, *rd = nullptr, *x = nullptr, *x2 = nullptr, *b = nullptr, *d = nullptr;
    double* tb = nullptr;   // right-hand side of the single-step entry points.  The cycle's own b of a coarse level is written ONLY by
                            // the restriction kernels: slots of coarse points under no fine tile are never written and must stay 0.
};

}  // namespace

namespace mgb {
void set_last_error(const std::string& msg) { g_last_error = msg; }
}  // namespace mgb

struct mg_handle_s {
    HostHierarchy hh;
    int L = 0;
    int solver = 0;                       // outer solver: 0 fGMRES(m), 1 BiCGStab
    double* bv[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // BiCGStab: rhat, p, v, s, t, y, z
    int P = 1;                            // planes solved together on this mesh; vectors are [plane][slot]
    int nu_pre = 2, nu_post = 2, m = 30, max_iters = 200;
    int gamma = 1;                        // cycle type: 1 V-cycle, 2 W-cycle, 3 F-cycle
    bool full_cgs2 = false;               // MG_SETUP_FULL_CGS2
    int64_t n = 0;
    std::vector<LevelDev> lev;
    LevelDev* d_lev = nullptr;            // device copy of lev[] (fused small-level kernel)
    int tail_s0 = 1 << 30;                // first level handled by the fused small-level kernel
    int tail_cap = 0;                     // its largest admissible grid
    std::vector<LevelBuf> buf;
    std::vector<void*> allocs;
    int32_t* user2slot = nullptr;
    // Krylov space (level-0 tile layout, stride = nslots of level 0)
    double *V = nullptr, *Z = nullptr, *w = nullptr, *r = nullptr, *xs = nullptr, *bs = nullptr;
    GmresState* st = nullptr;
    double* partial = nullptr;
    int* h_hdr = nullptr;                 // pinned copy of the first 8 ints of every plane's state (two slots of P x 8 ints)
    int* h_flag = nullptr;                // pinned copy of the coefficient flag (behind the headers)
    int* coeff_bad = nullptr;             // device flag of the last update: bit 0 lambda not finite, bit 1 c, bit 2 xi not finite or <= 0
    bool coeffs_unchecked = false;        // the flag of the last update has not been read yet (first solve / cycle after it)
    GmresState* h_state = nullptr;        // pinned full copy (read at the end of a solve)
    // coarsest level
    int nL = 0;
    int32_t *cslot = nullptr, *slot2row = nullptr;
    double *cwork = nullptr, *Ainv = nullptr;
    // host-buffer staging
    double* stage[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // lambda, c, x out, f, x0
    cudaStream_t copy_stream = nullptr;   // H2D of f, x0 overlaps the update's kernels (mg_solve_host)
    cudaEvent_t copy_ev = nullptr;
    double* stage_xi = nullptr;
    bool three_field = false;             // the level structs carry xi (Eq. 3)
    bool have_coeffs = false;
    bool no_fused_dr = false;             // debugging: separate defect + restriction kernel
    cudaError_t tail_err = cudaSuccess;
    bool host_only = false;
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t iter_graph = nullptr;
    int64_t iter_graph_kernels = 0;
    int64_t launches = 0;
    mg_alloc_fn alloc = nullptr;          // allocator installed when the handle was created: used for every later allocation
    mg_free_fn free_fn = nullptr;         // of this handle and by mg_destroy, whatever mg_set_allocator is called with afterwards
    int device = 0;
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // solve, update, single step
    cudaEvent_t hev[2] = {nullptr, nullptr};   // header copies of the two Arnoldi steps in flight
    bool solve_timed = false, update_timed = false, step_timed = false;
};

namespace {

int dev_alloc(mg_handle h, void** p, size_t bytes, cudaStream_t s) {
    *p = nullptr;
    if (bytes == 0) bytes = 8;
    if (h->alloc) {
        *p = h->alloc((uint64_t)bytes, (void*)s);
        if (!*p) { g_last_error = "allocator returned NULL"; return MG_ENOMEM; }
    } else {
        cudaError_t e = cudaMalloc(p, bytes);
        if (e != cudaSuccess) { g_last_error = std::string("cudaMalloc: ") + cudaGetErrorString(e); cudaGetLastError(); return MG_ENOMEM; }
    }
    h->allocs.push_back(*p);
    CU(cudaMemsetAsync(*p, 0, bytes, s));
    return MG_OK;
}

template <class T>
int upload(mg_handle h, T** dst, const std::vector<T>& src, cudaStream_t s) {
    int rc = dev_alloc(h, (void**)dst, src.size() * sizeof(T), s);
    if (rc) return rc;
    if (!src.empty()) CU(cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s));
    return MG_OK;
}

Launch LZ(mg_handle h, cudaStream_t s) { Launch L{s, &h->launches}; L.planes = h->P; return L; }
Launch LZ1(mg_handle h, cudaStream_t s) { return Launch{s, &h->launches}; }       // plane 0 only (single-step entry points)
VecRef lvec(mg_handle h, int level, double* p) { return vec(p, h->lev[level].nslots); }   // a level vector of all planes

// The last update's device-side admissibility flag (G26), already copied to *h_flag: MG_ECOEFF with the reason.
int coeff_error(int b) {
    g_last_error = std::string("inadmissible coefficients in the last update:") + ((b & 1) ? " lambda not finite;" : "") +
                   ((b & 2) ? " c not finite or <= 0 (PAPER.md:51);" : "") + ((b & 4) ? " xi not finite or <= 0;" : "") +
                   ((b & 8) ? " the coarsest-level operator is singular (zero or non-finite pivot);" : "");
    return MG_ECOEFF;
}

// Single-step entry points: read the flag of an update that has not been checked yet (one small synchronous copy).
int check_coeffs(mg_handle h, cudaStream_t s) {
    if (h->coeffs_unchecked) {
        CU(cudaMemcpyAsync(h->h_flag, h->coeff_bad, sizeof(int), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        h->coeffs_unchecked = false;
    }
    return *h->h_flag ? coeff_error(*h->h_flag) : MG_OK;
}

// nu Gauss-Seidel sweeps, two per launch where possible, ping-ponging between `cur` and `other`.
// Returns the buffer that holds the result.
// With `coarse`, the last launch also writes the restricted defect of the result to d_coarse; with `w_out`, A times the result.
VecRef enqueue_smooth(const Launch& L, const LevelDev& lv, VecRef cur, VecRef other, VecRef b, int nu, bool cur_is_zero,
                      const LevelDev* coarse = nullptr, double* d_coarse = nullptr, double* w_out = nullptr) {
    while (nu > 0) {
        const int k = nu >= 2 ? 2 : 1;
        launch_gs_fused(L, lv, cur, other, b, k, cur_is_zero, nu == k ? coarse : nullptr, d_coarse, nu == k ? w_out : nullptr);
        std::swap(cur, other);
        cur_is_zero = false;
        nu -= k;
    }
    return cur;
}

// Types of the visits a cycle of type `kind` (1 V, 2 W, 3 F) pays to the next coarser level: V: one V;
// W: two W; F: one F, then one V (the F-cycle of the paper's ref. [33], named at P:258; G24).
int cycle_visits(int kind, int out[2]) {
    if (kind == 2) { out[0] = out[1] = 2; return 2; }
    if (kind == 3) { out[0] = 3; out[1] = 1; return 2; }
    out[0] = 1;
    return 1;
}

// The same schedule as enqueue_cycle below, written as a program for the fused small-level kernel.
void build_tail(mg_handle h, int s, double* x, double* b, bool x_is_zero, TailProgram& P, int kind) {
    auto push = [&](TailOp op) { if (P.nops < TAIL_MAX_OPS) P.op[P.nops] = op; P.nops++; };
    const LevelDev& lv = h->lev[s];
    if (s == h->L - 1) { TailOp op{}; op.type = TAIL_COARSE; op.level = (unsigned char)s; op.ntiles = 1; op.a = b; op.b = x; push(op); return; }
    double *cur = x, *other = h->buf[s].x2;
    auto gs = [&](int k, int pc, bool zero, const double* ec) {
        TailOp op{}; op.type = TAIL_GS; op.level = (unsigned char)s; op.ns = (unsigned char)k; op.pc = (unsigned char)pc; op.zero = zero;
        op.ntiles = lv.ntiles; op.a = cur; op.b = other; op.c = b; op.ec = ec; op.dc = h->buf[s + 1].b; push(op);
        std::swap(cur, other);
    };
    const bool fuse_dr = !h->no_fused_dr;
    for (int nu = h->nu_pre; nu > 0;) { const int k = nu >= 2 ? 2 : 1; gs(k, (fuse_dr && nu == k) ? 2 : 0, x_is_zero, nullptr); x_is_zero = false; nu -= k; }
    if (!fuse_dr) { TailOp op{}; op.type = TAIL_DR; op.level = (unsigned char)s; op.ntiles = h->lev[s + 1].ntiles; op.a = cur; op.b = h->buf[s + 1].b; op.c = b; push(op); }
    int vk[2];
    const int nvis = cycle_visits(kind, vk);
    for (int g = 0; g < nvis; g++) build_tail(h, s + 1, h->buf[s + 1].x, h->buf[s + 1].b, g == 0, P, vk[g]);
    int nu = h->nu_post;
    { const int k = nu >= 2 ? 2 : 1; gs(k, 1, false, h->buf[s + 1].x); nu -= k; }
    while (nu > 0) { const int k = nu >= 2 ? 2 : 1; gs(k, 0, false, nullptr); nu -= k; }
    if (cur != x) { TailOp op{}; op.type = TAIL_COPY; op.level = (unsigned char)s; op.a = cur; op.b = x; op.n = lv.nslots; push(op); }
}

// mg_cycle of PAPER.md:171-195 (cycle type `kind`, 0 = the handle's), enqueued on L.stream.  x_is_zero: the initial guess is
// the zero vector and x need not be read (nor zeroed beforehand).  w_out: also produce w_out = A x for the
// result (fused into the last smoothing launch); returns whether it was written.
bool enqueue_cycle(mg_handle h, const Launch& L, int s, VecRef x, VecRef b, bool x_is_zero, double* w_out = nullptr, int kind = 0) {
    const LevelDev& lv = h->lev[s];
    if (kind == 0) kind = h->gamma;
    if (s >= h->tail_s0 && h->P == 1) {                                            // small levels: one cooperative kernel
        TailProgram P; P.nops = 0;
        build_tail(h, s, TAIL_TOPX, TAIL_TOPB, x_is_zero, P, kind);
        if (P.nops <= TAIL_MAX_OPS) {
            int grid = 1;
            for (int i = 0; i < P.nops; i++) grid = std::max(grid, P.op[i].type == TAIL_COPY ? 8 : P.op[i].ntiles);
            TailCoarse cs{h->Ainv, h->cslot, h->nL};
            if (grid <= h->tail_cap && h->L - s <= TAIL_MAX_LEVELS) {
                h->tail_err = launch_tail(L, h->d_lev, s, h->L, P, cs, x, b, grid);
                return false;
            }
        }
    }
    if (s == h->L - 1) {                                              // P:173-177 direct solve
        launch_coarse_solve(L, h->Ainv, h->cslot, h->nL, b, x);
        return false;
    }
    VecRef tmp = lvec(h, s, h->buf[s].x2);
    if (x_is_zero && h->nu_pre == 0) { launch_zero(L, x, lv.nslots); x_is_zero = false; }
    const bool fuse_dr = h->nu_pre > 0 && !h->no_fused_dr;
    VecRef cur = enqueue_smooth(L, lv, x, tmp, b, h->nu_pre, x_is_zero,                   // P:178-181 (+ P:183-184 fused)
                                fuse_dr ? &h->lev[s + 1] : nullptr, h->buf[s + 1].b);
    VecRef other = (cur.base == x.base) ? tmp : x;
    if (!fuse_dr) launch_defect_restrict(L, lv, h->lev[s + 1], cur, b, h->buf[s + 1].b);  // P:183-184  R (A x - b)
    int vk[2];
    const int nvis = cycle_visits(kind, vk);
    for (int g = 0; g < nvis; g++)                                                        // e0 = 0, gamma visits
        enqueue_cycle(h, L, s + 1, lvec(h, s + 1, h->buf[s + 1].x), lvec(h, s + 1, h->buf[s + 1].b), g == 0, nullptr, vk[g]);
    VecRef fin;
    bool wrote_w = false;
    if (h->nu_post > 0) {                                 // P:194-197 fused into the first post-smoothing pass
        const int k = h->nu_post >= 2 ? 2 : 1, rem = h->nu_post - k;
        launch_gs_correct(L, lv, h->buf[s + 1].x, cur, other, b, k, rem == 0 ? w_out : nullptr);
        fin = enqueue_smooth(L, lv, other, cur, b, rem, false, nullptr, nullptr, w_out);
        wrote_w = w_out != nullptr;
    } else {
        launch_prolong_correct(L, lv, h->lev[s + 1], h->buf[s + 1].x, h->buf[s].d, cur);
        fin = cur;
    }
    if (fin.base != x.base) launch_copy(L, fin, x, lv.nslots);
    return wrote_w;
}

// One Arnoldi step (rule K2): z_j = MG(v_j), w = A z_j, CGS2, Givens + stop test, v_{j+1}.
void enqueue_iteration(mg_handle h, const Launch& L) {
    const int64_t ns = h->lev[0].nslots;
    const int64_t bps = (int64_t)(h->m + 1) * ns;                    // plane stride of the Krylov bases
    VecRef zj{h->Z, ns, &h->st->j, 0, bps}, vj{h->V, ns, &h->st->j, 0, bps};
    static const bool no_fused_apply = getenv("MG_B200_NO_FUSED_APPLY") != nullptr;
    if (!enqueue_cycle(h, L, 0, zj, vj, true, no_fused_apply ? nullptr : h->w))          // w = A z_j fused into the cycle's last launch
        launch_apply(L, h->lev[0], zj, vec(nullptr), vec(h->w, ns), 0);
    launch_multidot(L, h->w, h->V, ns, ns, h->st, h->partial, h->m);
    if (h->m <= MAX_M_FUSED) {                                     // three passes over the basis
        launch_update_dot(L, h->w, h->V, ns, ns, h->st, h->partial);
        launch_final_v(L, h->w, h->V, ns, ns, h->st);
        return;
    }
    launch_update_w(L, h->w, h->V, ns, ns, h->st, h->partial, 0);
    launch_multidot(L, h->w, h->V, ns, ns, h->st, h->partial, h->m);
    launch_update_w(L, h->w, h->V, ns, ns, h->st, h->partial, 1);
    launch_givens(L, h->st);
    launch_next_v(L, h->w, h->V, ns, ns, h->st);
}

// One BiCGStab step (mg_bicgstab.cu): two preconditioner applications, each with its operator apply fused into the
// cycle's last smoothing launch; the second application is skipped on the device after a half step.
void enqueue_bicgstab_step(mg_handle h, const Launch& L) {
    const int64_t ns = h->lev[0].nslots;
    double *rhat = h->bv[0], *p = h->bv[1], *v = h->bv[2], *sv = h->bv[3], *t = h->bv[4], *y = h->bv[5], *z = h->bv[6];
    launch_bi_p(L, h->st, h->r, p, v, ns);
    if (!enqueue_cycle(h, L, 0, vec(y, ns), vec(p, ns), true, v)) launch_apply(L, h->lev[0], vec(y, ns), vec(nullptr), vec(v, ns), 0);
    launch_bi_alpha(L, h->st, rhat, v, ns, h->partial);
    launch_bi_s(L, h->st, h->r, v, sv, ns, h->partial);
    Launch L2 = L;
    L2.stop = &h->st->b_skip2;                            // z = M s, t = A z: not after a half step
    if (!enqueue_cycle(h, L2, 0, vec(z, ns), vec(sv, ns), true, t)) launch_apply(L2, h->lev[0], vec(z, ns), vec(nullptr), vec(t, ns), 0);
    launch_bi_omega(L, h->st, t, sv, ns, h->partial);
    launch_bi_update(L, h->st, h->xs, h->r, rhat, y, z, sv, t, ns, h->partial);
}

int build_iter_graph(mg_handle h) {
    if (h->iter_graph) return MG_OK;
    cudaGraph_t g = nullptr;
    const int64_t before = h->launches;
    CU(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    Launch L = LZ(h, h->cap_stream);
    L.stop = &h->st->cycle_end;          // iterations are enqueued one ahead of the convergence test
    if (h->solver == 1) enqueue_bicgstab_step(h, L); else enqueue_iteration(h, L);
    CU(cudaStreamEndCapture(h->cap_stream, &g));
    CU(h->tail_err);
    h->iter_graph_kernels = h->launches - before;
    h->launches = before;
    CU(cudaGraphInstantiate(&h->iter_graph, g, 0));
    CU(cudaGraphDestroy(g));
    return MG_OK;
}

}  // namespace

extern "C" {

const char* mg_last_error(void) { return g_last_error.c_str(); }

const char* mg_strerror(int code) {
    switch (code) {
        case MG_OK: return "ok";
        case MG_NOT_CONVERGED: return "not converged (max_iters reached)";
        case MG_BREAKDOWN: return "breakdown (h_{j+1,j} = 0)";
        case MG_EINVAL: return "invalid argument";
        case MG_EMESH: return "invalid mesh";
        case MG_ECOEFF: return "invalid coefficients";
        case MG_ENOTREADY: return "mg_update_coeffs has not been called";
        case MG_ECUDA: return "CUDA error";
        case MG_ENOMEM: return "out of device memory";
        default: return "unknown error";
    }
}

int mg_set_allocator(mg_alloc_fn a, mg_free_fn f) {
    if ((a == nullptr) != (f == nullptr)) return MG_EINVAL;
    g_alloc = a; g_free = f;
    return MG_OK;
}

int mg_destroy(mg_handle h) {
    if (!h) return MG_EINVAL;
    if (h->host_only) { delete h; return MG_OK; }
    cudaDeviceSynchronize();
    if (h->iter_graph) cudaGraphExecDestroy(h->iter_graph);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    if (h->copy_ev) cudaEventDestroy(h->copy_ev);
    for (auto& e : h->ev) if (e) cudaEventDestroy(e);
    for (auto& e : h->hev) if (e) cudaEventDestroy(e);
    if (h->h_hdr) cudaFreeHost(h->h_hdr);
    if (h->h_state) cudaFreeHost(h->h_state);
    for (void* p : h->allocs) { if (h->free_fn) h->free_fn(p); else cudaFree(p); }
    delete h;
    return MG_OK;
}

int mg_setup(const mg_mesh* mesh, const mg_bc* bc, const mg_options* opt, void* stream, mg_handle* out) {
    if (!out) return MG_EINVAL;
    *out = nullptr;
    if (!mesh || !bc || !mesh->i || !mesh->j || !bc->kind || mesh->n <= 0 || !(mesh->h > 0.0)) { g_last_error = "null pointer, n <= 0 or h <= 0"; return MG_EINVAL; }
    mg_options o{};
    if (opt) o = *opt;
    if (o.levels < 0 || o.nu_pre < 0 || o.nu_post < MG_NU_NONE || o.restart_m < 0 || o.restart_m > MAX_M || o.max_iters < 0 || o.gamma < 0 || o.gamma > 3 || (o.flags & ~7) != 0 || o.planes < 0 || o.planes > 4096 || o.solver < 0 || o.solver > 1) { g_last_error = "bad option"; return MG_EINVAL; }
    const bool host_only = (o.flags & 1) != 0;
    int ndev = 0;
    if (!host_only && (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)) { cudaGetLastError(); g_last_error = "no CUDA device (this library has no CPU fallback)"; return MG_ECUDA; }
    mg_handle h = new (std::nothrow) mg_handle_s();
    if (!h) return MG_ENOMEM;
    h->nu_pre = o.nu_pre ? o.nu_pre : 2;
    h->nu_post = o.nu_post == 0 ? 2 : (o.nu_post == MG_NU_NONE ? 0 : o.nu_post);
    h->m = o.restart_m ? o.restart_m : 30;
    h->max_iters = o.max_iters ? o.max_iters : 200;
    h->gamma = o.gamma > 1 ? o.gamma : 1;
    h->P = o.planes > 1 ? o.planes : 1;
    h->solver = o.solver;
    h->full_cgs2 = (o.flags & MG_SETUP_FULL_CGS2) != 0;
    h->n = mesh->n;
    h->alloc = g_alloc; h->free_fn = g_free;
    int rc = build_hierarchy(mesh->n, mesh->i, mesh->j, bc->kind, mesh->h, o.levels, h->hh);
    if (rc) { g_last_error = h->hh.err; delete h; return rc; }
    h->L = (int)h->hh.lev.size();
    h->nL = (int)h->hh.lev.back().n;
    if (h->nL > 1024) { g_last_error = "coarsest level has more than 1024 points; use more levels"; delete h; return MG_EMESH; }
    if (host_only) { h->host_only = true; *out = h; return MG_OK; }
    cudaStream_t s = (cudaStream_t)stream;
    cudaGetDevice(&h->device);
    auto fail = [&](int code) { mg_destroy(h); return code; };
#define TRY(x) do { int rc__ = (x); if (rc__) return fail(rc__); } while (0)
#define CUF(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { g_last_error = std::string(#call) + ": " + cudaGetErrorString(e__); return fail(MG_ECUDA); } } while (0)
    CUF(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    for (auto& e : h->ev) CUF(cudaEventCreate(&e));
    for (auto& e : h->hev) CUF(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    CUF(cudaMallocHost((void**)&h->h_hdr, sizeof(int) * (16 * (size_t)h->P + 8)));      // two header slots of 8 ints per plane + the coefficient flag
    h->h_flag = h->h_hdr + 16 * (size_t)h->P;
    *h->h_flag = 0;
    TRY(dev_alloc(h, (void**)&h->coeff_bad, sizeof(int), s));
    CUF(cudaMallocHost((void**)&h->h_state, sizeof(GmresState) * h->P));
    h->lev.resize(h->L); h->buf.resize(h->L);
    for (int l = 0; l < h->L; l++) {
        HostLevel& hl = h->hh.lev[l];
        LevelBuf& b = h->buf[l];
        TRY(upload(h, &b.code, hl.code, s));
        TRY(upload(h, &b.tnb, hl.tnb, s));
        TRY(upload(h, &b.tflag, hl.tflag, s));
        TRY(upload(h, &b.ctab, hl.ctab, s));
        TRY(upload(h, &b.ptab, hl.ptab, s));
        std::vector<int32_t> tij(2 * (size_t)hl.ntiles);
        for (int t = 0; t < hl.ntiles; t++) { tij[2 * t] = hl.tI[t]; tij[2 * t + 1] = hl.tJ[t]; }
        TRY(upload(h, &b.tij, tij, s));
        TRY(upload(h, &b.canon2slot, hl.canon2slot, s));
        for (int k = 0; k < 2; k++) {
            TRY(upload(h, &b.tlist[k], hl.tlist[k], s));
            const int32_t nmeta = hl.nint[k] + hl.ngen[k];
            std::vector<int32_t> meta((size_t)24 * nmeta, 0);                // tables of the interior and general tiles, packed in list order
            for (int32_t q = 0; q < nmeta; q++) {
                const int32_t t = hl.tlist[k][q];
                for (int e = 0; e < 9; e++) { meta[24 * (size_t)q + e] = hl.tnb[9 * (size_t)t + e]; meta[24 * (size_t)q + 9 + e] = hl.ptab.empty() ? 0 : hl.ptab[9 * (size_t)t + e]; }
                meta[24 * (size_t)q + 18] = hl.tI[t] & 1; meta[24 * (size_t)q + 19] = hl.tJ[t] & 1; meta[24 * (size_t)q + 20] = t;
            }
            TRY(upload(h, &b.smeta[k], meta, s));
        }
        const size_t vb1 = (size_t)hl.nslots() * sizeof(double), vb = vb1 * h->P;      // every vector once per plane
        TRY(dev_alloc(h, (void**)&b.lam, vb, s));
        TRY(dev_alloc(h, (void**)&b.c, vb, s));
        TRY(dev_alloc(h, (void**)&b.rd, vb, s));
        TRY(dev_alloc(h, (void**)&b.x, vb, s));
        TRY(dev_alloc(h, (void**)&b.x2, vb, s));
        TRY(dev_alloc(h, (void**)&b.b, vb, s));
        TRY(dev_alloc(h, (void**)&b.d, vb, s));
        TRY(dev_alloc(h, (void**)&b.tb, vb1, s));
        LevelDev& d = h->lev[l];
        d.ntiles = hl.ntiles;
        d.ntiles_fine = l > 0 ? h->hh.lev[l - 1].ntiles : 0;
        d.ntiles_coarse = l + 1 < h->L ? h->hh.lev[l + 1].ntiles : 0;
        d.nslots = hl.nslots();
        d.h = hl.h; d.kappa = 1.0 / (2.0 * hl.h * hl.h);
        d.code = b.code; d.tnb = b.tnb; d.ctab = b.ctab; d.ptab = b.ptab; d.tij = b.tij; d.lam = b.lam; d.c = b.c; d.rd = b.rd; d.tflag = b.tflag;
        d.xi = nullptr;
        for (int k = 0; k < 2; k++) { d.tlist[k] = b.tlist[k]; d.nint[k] = hl.nint[k]; d.ngen[k] = hl.ngen[k]; d.smeta[k] = b.smeta[k]; }
    }
    TRY(dev_alloc(h, (void**)&h->d_lev, sizeof(LevelDev) * h->L, s));
    CUF(cudaMemcpyAsync(h->d_lev, h->lev.data(), sizeof(LevelDev) * h->L, cudaMemcpyHostToDevice, s));
    h->no_fused_dr = getenv("MG_B200_NO_FUSED_DR") != nullptr;
    h->tail_cap = std::min(tail_max_grid(), 2 * dev_info().sms);
    if (h->P == 1 && h->tail_cap > 0 && h->nu_pre >= 1 && h->nu_post >= 1 && ((o.flags & MG_SETUP_FUSED_TAIL) || getenv("MG_B200_FUSED_TAIL")))
        for (int l = h->L - 1; l >= 0 && h->lev[l].ntiles <= h->tail_cap; l--) h->tail_s0 = l;
    TRY(upload(h, &h->user2slot, h->hh.user2slot, s));
    const size_t v0 = (size_t)h->lev[0].nslots * sizeof(double) * h->P;
    if (h->solver == 0) {
        TRY(dev_alloc(h, (void**)&h->V, v0 * (h->m + 1), s));
        TRY(dev_alloc(h, (void**)&h->Z, v0 * (h->m + 1), s));
    } else {
        for (int k = 0; k < 7; k++) TRY(dev_alloc(h, (void**)&h->bv[k], v0, s));     // no Krylov basis: seven work vectors
    }
    TRY(dev_alloc(h, (void**)&h->w, v0, s));
    TRY(dev_alloc(h, (void**)&h->r, v0, s));
    TRY(dev_alloc(h, (void**)&h->xs, v0, s));
    TRY(dev_alloc(h, (void**)&h->bs, v0, s));
    TRY(dev_alloc(h, (void**)&h->st, sizeof(GmresState) * h->P, s));
    TRY(dev_alloc(h, (void**)&h->partial, sizeof(double) * RED_BLOCKS_MAX * (MAX_M + 2) * h->P, s));
    {   // coarsest level: canonical row -> slot and its inverse
        HostLevel& cl = h->hh.lev.back();
        std::vector<int32_t> s2r((size_t)cl.nslots(), 0);
        for (int r = 0; r < h->nL; r++) s2r[cl.canon2slot[r]] = r;
        h->cslot = h->buf[h->L - 1].canon2slot;
        TRY(upload(h, &h->slot2row, s2r, s));
        TRY(dev_alloc(h, (void**)&h->cwork, sizeof(double) * coarse_work_doubles(h->nL) * h->P, s));   // [A | I] + published column (x2) + pivots
        TRY(dev_alloc(h, (void**)&h->Ainv, sizeof(double) * (size_t)h->nL * h->nL * h->P, s));
    }
    CUF(cudaStreamSynchronize(s));
#undef TRY
#undef CUF
    *out = h;
    return MG_OK;
}

}  // extern "C"

// ============================================================================ update / solve
extern "C" {

// Switch the level structs between the two-field (xi null) and the three-field form.  The structs are kernel
// arguments baked into the captured iteration graph and copied to the device for the fused small-level kernel, so
// both are refreshed.
static int set_three_field(mg_handle h, bool on, cudaStream_t s) {
    if (h->three_field == on) return MG_OK;
    for (int l = 0; l < h->L; l++) {
        LevelBuf& b = h->buf[l];
        if (on && !b.xi) {
            const size_t vb = (size_t)h->hh.lev[l].nslots() * sizeof(double) * h->P;
            int rc = dev_alloc(h, (void**)&b.xi, vb, s); if (rc) return rc;
        }
        h->lev[l].xi = on ? b.xi : nullptr;
    }
    CU(cudaStreamSynchronize(s));         // h->lev is pageable host memory: the copy below must not overlap a later change
    CU(cudaMemcpyAsync(h->d_lev, h->lev.data(), sizeof(LevelDev) * h->L, cudaMemcpyHostToDevice, s));
    CU(cudaStreamSynchronize(s));
    if (h->iter_graph) { cudaGraphExecDestroy(h->iter_graph); h->iter_graph = nullptr; }
    h->three_field = on;
    return MG_OK;
}

int mg_update_coeffs3(mg_handle h, const double* d_lambda, const double* d_xi, const double* d_c, void* stream) {
    if (!h || !d_lambda || !d_c) return MG_EINVAL;
    if (h->host_only) return MG_ECUDA;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = set_three_field(h, d_xi != nullptr, s);
    if (rc) return rc;
    Launch L = LZ(h, s);
    CU(cudaEventRecord(h->ev[2], s));
    // admissibility (c > 0; lambda only finite since Eq. 21 P:241 has both signs; xi > 0, G25) is tested on the device while
    // the fields are gathered; the first mg_solve after the update reads the flag and returns MG_ECOEFF
    CU(cudaMemsetAsync(h->coeff_bad, 0, sizeof(int), s));
    const int64_t ns0 = h->lev[0].nslots;
    launch_gather_check(L, d_lambda, h->user2slot, h->buf[0].lam, h->n, ns0, 1, 1, h->coeff_bad);
    launch_gather_check(L, d_c, h->user2slot, h->buf[0].c, h->n, ns0, 2, 2, h->coeff_bad);
    if (d_xi) launch_gather_check(L, d_xi, h->user2slot, h->buf[0].xi, h->n, ns0, 2, 4, h->coeff_bad);
    h->coeffs_unchecked = true;
    for (int l = 0; l + 1 < h->L; l++) launch_restrict_coeff(L, h->lev[l], h->lev[l + 1]);     // rule T4
    for (int l = 0; l < h->L; l++) launch_diag(L, h->lev[l]);                                   // U2: 1 / a_ll for the smoother
    launch_coarse_factor(L, h->lev[h->L - 1], h->cslot, h->slot2row, h->nL, h->cwork, h->Ainv, h->coeff_bad);   // rule C
    CU(cudaEventRecord(h->ev[3], s));
    CU(cudaGetLastError());
    h->have_coeffs = true;
    h->update_timed = true;
    return MG_OK;
}

int mg_update_coeffs(mg_handle h, const double* d_lambda, const double* d_c, void* stream) {
    return mg_update_coeffs3(h, d_lambda, nullptr, d_c, stream);
}

// first 8 ints (j, iters, status, cycle_end, ...) of every plane's state -> pinned header slot `slot`
static int copy_headers(mg_handle h, int slot, cudaStream_t s) {
    CU(cudaMemcpy2DAsync(h->h_hdr + (size_t)slot * 8 * h->P, 32, h->st, sizeof(GmresState), 32, h->P, cudaMemcpyDeviceToHost, s));
    return MG_OK;
}
static bool all_ended(mg_handle h, int slot) {
    for (int p = 0; p < h->P; p++) if (!h->h_hdr[((size_t)slot * h->P + p) * 8 + 3]) return false;
    return true;
}

int mg_solve(mg_handle h, const double* d_f, const double* d_x0, double* d_x, double rtol, int* iters,
             double* final_relres, void* stream) {
    if (!h || !d_f || !d_x0 || !d_x || !(rtol > 0.0)) return MG_EINVAL;
    if (h->host_only) return MG_ECUDA;
    if (!h->have_coeffs) return MG_ENOTREADY;
    cudaStream_t s = (cudaStream_t)stream;
    Launch L = LZ(h, s);
    int rc = build_iter_graph(h);
    if (rc) return rc;
    const int64_t ns = h->lev[0].nslots;
    const int P = h->P;
    CU(cudaEventRecord(h->ev[0], s));
    launch_init_state(L, h->st, h->m, h->max_iters, rtol, h->full_cgs2);
    launch_gather(L, d_f, h->user2slot, h->bs, h->n, ns);             // B1: user order -> tile layout
    launch_gather(L, d_x0, h->user2slot, h->xs, h->n, ns);
    launch_norm2(L, h->bs, ns, h->st, h->partial, 0);                 // K1: bn = ||b||
    // All planes run the same launches; each has its own state.  A plane whose restart cycle has ended (converged,
    // m columns, max_iters, breakdown) makes its CTAs return at once until every plane has ended the cycle; then
    // x is updated (a plane that did not start the cycle adds nothing) and the next cycle starts where needed.
    for (int cycle = 0; cycle < 1000000; cycle++) {
        launch_apply(L, h->lev[0], vec(h->xs, ns), vec(h->bs, ns), vec(h->r, ns), 1);      // r = b - A x (rule D4)
        launch_norm2(L, h->r, ns, h->st, h->partial, 1);
        if (h->solver == 1) launch_bi_start(L, h->st, h->r, h->bv[0], ns);
        else launch_start_cycle(L, h->st, h->r, h->V, ns);
        rc = copy_headers(h, 0, s);
        if (rc) return rc;
        if (h->coeffs_unchecked) CU(cudaMemcpyAsync(h->h_flag, h->coeff_bad, sizeof(int), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        h->coeffs_unchecked = false;
        if (*h->h_flag) {                                             // the last update's fields were not admissible
            h->solve_timed = false;                                   // ev[0] has no matching end event
            return coeff_error(*h->h_flag);
        }
        if (all_ended(h, 0)) break;                                   // no plane started a cycle: finished
        // One graph launch per Arnoldi step.  The host stays one step ahead: step `it` is enqueued before
        // the headers of step it-1 are inspected, so the GPU never idles on the round trip; a step enqueued
        // after the cycle has ended finds cycle_end set and every kernel in it returns at once.
        const int nsteps = h->solver == 1 ? h->max_iters / 2 + 2 : h->m;      // BiCGStab: no restart length, the cap ends the cycle
        for (int it = 0; it < nsteps; it++) {
            CU(cudaGraphLaunch(h->iter_graph, s));
            h->launches += h->iter_graph_kernels;
            rc = copy_headers(h, it & 1, s);
            if (rc) return rc;
            CU(cudaEventRecord(h->hev[it & 1], s));
            if (it >= 1) {
                CU(cudaEventSynchronize(h->hev[(it - 1) & 1]));
                if (all_ended(h, (it - 1) & 1)) break;
            }
        }
        if (h->solver == 0) launch_update_x(L, h->xs, h->Z, ns, ns, h->st);               // K4 (BiCGStab updates x in place)
    }
    launch_zero_rhs_planes(L, h->xs, ns, h->st);                      // K1: zero right-hand side -> x = 0
    launch_scatter(L, h->xs, h->user2slot, d_x, h->n, ns);            // B1: tile layout -> user order
    CU(cudaEventRecord(h->ev[1], s));
    CU(cudaMemcpyAsync(h->h_state, h->st, sizeof(GmresState) * P, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    CU(cudaGetLastError());
    h->solve_timed = true;
    int worst = MG_OK;                                                // over the planes: breakdown > not converged > ok
    for (int p = 0; p < P; p++) {
        const GmresState* st = &h->h_state[p];
        if (iters) iters[p] = st->iters;
        if (final_relres) final_relres[p] = st->relres;
        const int r1 = (st->status == 1 || st->status == 4) ? MG_OK : (st->status == 3 ? MG_BREAKDOWN : MG_NOT_CONVERGED);
        if (r1 == MG_NOT_CONVERGED) {
            // If the recurrence residual (Eq. 23 inside a cycle, rule K3) went below rtol while the recomputed true residual
            // (rule K5) did not, the solve sits on the fp64 floor of evaluating b - A x, about eps |A||x| / |b| ~ 1/h^2
            // (DESIGN.md "Attainable accuracy"); the paper has no stagnation exit, so the call only says so.
            const int k = std::min(st->iters, 512);
            double best = 1e300;
            for (int i = 0; i < k; i++) best = std::min(best, st->hist[i]);
            char buf[360];
            if (k > 0 && best < rtol)
                snprintf(buf, sizeof buf, "plane %d not converged after %d iterations: the recurrence residual reached %.2e < rtol = %.2e but the true "
                         "residual |b - A x| / |b| stays at %.2e: rtol is below the accuracy attainable in fp64 on this mesh", p, st->iters, best, rtol, st->relres);
            else
                snprintf(buf, sizeof buf, "plane %d not converged after %d iterations: |b - A x| / |b| = %.2e, rtol = %.2e", p, st->iters, st->relres, rtol);
            g_last_error = buf;
        }
        worst = std::max(worst, r1);
    }
    return worst;
}

static int ensure_stage(mg_handle h, cudaStream_t s) {
    for (int k = 0; k < 5; k++)
        if (!h->stage[k]) { int rc = dev_alloc(h, (void**)&h->stage[k], sizeof(double) * (size_t)h->n * h->P, s); if (rc) return rc; }
    return MG_OK;
}

int mg_update_coeffs_host(mg_handle h, const double* h_lambda, const double* h_c, void* stream) {
    if (!h || !h_lambda || !h_c) return MG_EINVAL;
    if (h->host_only) return MG_ECUDA;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_stage(h, s);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->stage[0], h_lambda, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(h->stage[1], h_c, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, s));
    return mg_update_coeffs(h, h->stage[0], h->stage[1], stream);
}

int mg_update_coeffs3_host(mg_handle h, const double* h_lambda, const double* h_xi, const double* h_c, void* stream) {
    if (!h || !h_lambda || !h_c) return MG_EINVAL;
    if (!h_xi) return mg_update_coeffs_host(h, h_lambda, h_c, stream);
    if (h->host_only) return MG_ECUDA;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_stage(h, s);
    if (rc) return rc;
    if (!h->stage_xi) { rc = dev_alloc(h, (void**)&h->stage_xi, sizeof(double) * (size_t)h->n * h->P, s); if (rc) return rc; }
    CU(cudaMemcpyAsync(h->stage[0], h_lambda, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(h->stage[1], h_c, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(h->stage_xi, h_xi, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, s));
    return mg_update_coeffs3(h, h->stage[0], h->stage_xi, h->stage[1], stream);
}

int mg_solve_host(mg_handle h, const double* h_f, const double* h_x0, double* h_x, double rtol, int* iters,
                  double* final_relres, void* stream) {
    if (!h || !h_f || !h_x0 || !h_x) return MG_EINVAL;
    if (h->host_only) return MG_ECUDA;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = ensure_stage(h, s);
    if (rc) return rc;
    // f and x0 travel on their own stream into their own buffers: the copies need not wait for the update's kernels
    // (which are still reading the lambda / c staging buffers on `s`); the solve waits for the copies
    if (!h->copy_stream) { CU(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking)); CU(cudaEventCreateWithFlags(&h->copy_ev, cudaEventDisableTiming)); }
    CU(cudaMemcpyAsync(h->stage[3], h_f, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, h->copy_stream));
    CU(cudaMemcpyAsync(h->stage[4], h_x0, sizeof(double) * h->n * h->P, cudaMemcpyHostToDevice, h->copy_stream));
    CU(cudaEventRecord(h->copy_ev, h->copy_stream));
    CU(cudaStreamWaitEvent(s, h->copy_ev, 0));
    rc = mg_solve(h, h->stage[3], h->stage[4], h->stage[2], rtol, iters, final_relres, stream);
    if (rc < 0) return rc;
    CU(cudaMemcpyAsync(h_x, h->stage[2], sizeof(double) * h->n * h->P, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return rc;
}

int64_t mg_kernel_launches(mg_handle h) { return h ? h->launches : 0; }

int mg_last_history(mg_handle h, double* relres, double* orth, int cap) {
    if (!h || cap < 0) return MG_EINVAL;
    if (!h->solve_timed) return 0;
    const int n = std::min(std::min(h->h_state->iters, 512), cap);
    for (int k = 0; k < n; k++) {
        if (relres) relres[k] = h->h_state->hist[k];
        if (orth) orth[k] = h->h_state->orth[k];
    }
    return n;
}

int mg_last_reorth(mg_handle h) { return (h && h->solve_timed) ? h->h_state->nreorth : -1; }

double mg_last_solve_ms(mg_handle h) {
    float ms = -1.f;
    if (!h || !h->solve_timed || cudaEventElapsedTime(&ms, h->ev[0], h->ev[1]) != cudaSuccess) { cudaGetLastError(); return -1.0; }
    return ms;
}
double mg_last_step_ms(mg_handle h) {
    float ms = -1.f;
    if (!h || !h->step_timed || cudaEventSynchronize(h->ev[5]) != cudaSuccess || cudaEventElapsedTime(&ms, h->ev[4], h->ev[5]) != cudaSuccess) { cudaGetLastError(); return -1.0; }
    return ms;
}
double mg_last_update_ms(mg_handle h) {
    float ms = -1.f;
    if (!h || !h->update_timed || cudaEventSynchronize(h->ev[3]) != cudaSuccess || cudaEventElapsedTime(&ms, h->ev[2], h->ev[3]) != cudaSuccess) { cudaGetLastError(); return -1.0; }
    return ms;
}

}  // extern "C"

// ============================================================================ inspection
extern "C" {

int mg_num_levels(mg_handle h) { return h ? h->L : MG_EINVAL; }
int64_t mg_level_n(mg_handle h, int level) { return (h && level >= 0 && level < h->L) ? h->hh.lev[level].n : (int64_t)MG_EINVAL; }

int mg_level_info(mg_handle h, int level, int32_t* I, int32_t* J, uint8_t* kind, uint8_t* colour, int32_t* nbr,
                  int8_t* ns_tn, uint8_t* ns_fallback, int32_t* slot, int64_t* user2canon) {
    if (!h || level < 0 || level >= h->L) return MG_EINVAL;
    const HostLevel& lv = h->hh.lev[level];
    std::vector<int32_t> s2c;
    if (nbr || user2canon) {
        s2c.assign((size_t)lv.nslots(), -1);
        for (int64_t k = 0; k < lv.n; k++) s2c[lv.canon2slot[k]] = (int32_t)k;
    }
    const int dI[4] = {-1, 1, 0, 0}, dJ[4] = {0, 0, -1, 1};
    for (int64_t k = 0; k < lv.n; k++) {
        const int64_t s = lv.canon2slot[k];
        const int t = (int)(s / TS), ly = (int)(s % TS) / TX, lx = (int)(s % TS) % TX;
        const int64_t pi = (int64_t)lv.tI[t] * TX + lx, pj = (int64_t)lv.tJ[t] * TY + ly;
        const uint16_t c = lv.code[s];
        const int kd = code_kind(c);
        if (I) I[k] = (int32_t)pi;
        if (J) J[k] = (int32_t)pj;
        if (kind) kind[k] = (uint8_t)(kd - 1);
        if (colour) colour[k] = (uint8_t)(kd == C_INNER ? ((pi + pj) & 1) : 2);          // rule M6
        if (nbr)
            for (int d = 0; d < 4; d++) {
                const int64_t q = lv.slot_of(pi + dI[d], pj + dJ[d]);
                nbr[4 * k + d] = q < 0 ? -1 : s2c[q];
            }
        if (ns_tn) {
            ns_tn[2 * k] = (int8_t)(kd == C_NEU ? ((c >> 2) & 7) - 2 : 0);
            ns_tn[2 * k + 1] = (int8_t)(kd == C_NEU ? ((c >> 5) & 7) - 2 : 0);
        }
        if (ns_fallback) ns_fallback[k] = (uint8_t)(kd == C_NEU ? (c >> 8) & 1 : 0);
        if (slot) slot[k] = (int32_t)s;
    }
    if (user2canon) {
        if (level != 0) return MG_EINVAL;
        for (int64_t p = 0; p < h->n; p++) user2canon[p] = s2c[h->hh.user2slot[p]];
    }
    return MG_OK;
}

int mg_transfer_info(mg_handle h, int level, int32_t* fine9, int32_t* parent, uint8_t* ptype) {
    if (!h || level < 0 || level + 1 >= h->L) return MG_EINVAL;
    const HostLevel &f = h->hh.lev[level], &c = h->hh.lev[level + 1];
    auto s2c_of = [](const HostLevel& lv) {
        std::vector<int32_t> m((size_t)lv.nslots(), -1);
        for (int64_t k = 0; k < lv.n; k++) m[lv.canon2slot[k]] = (int32_t)k;
        return m;
    };
    auto coords = [](const HostLevel& lv, int64_t s, int64_t& pi, int64_t& pj) {
        const int t = (int)(s / TS);
        pi = (int64_t)lv.tI[t] * TX + (s % TS) % TX; pj = (int64_t)lv.tJ[t] * TY + (s % TS) / TX;
    };
    if (fine9) {
        const std::vector<int32_t> fm = s2c_of(f);
        for (int64_t q = 0; q < c.n; q++) {
            int64_t ci, cj; coords(c, c.canon2slot[q], ci, cj);
            for (int dy = -1; dy <= 1; dy++)
                for (int dx = -1; dx <= 1; dx++) {
                    const int64_t s = f.slot_of(2 * ci + dx, 2 * cj + dy);
                    fine9[9 * q + 3 * (dy + 1) + dx + 1] = s < 0 ? -1 : fm[s];
                }
        }
    }
    if (parent || ptype) {
        const std::vector<int32_t> cm = s2c_of(c);
        for (int64_t l = 0; l < f.n; l++) {
            int64_t fi, fj; coords(f, f.canon2slot[l], fi, fj);
            const int ox = (int)(fi & 1), oy = (int)(fj & 1);
            const int64_t ci = floordiv(fi, 2), cj = floordiv(fj, 2);
            if (ptype) ptype[l] = (uint8_t)(ox + 2 * oy);
            if (parent) {
                int cnt = 0;
                for (int b = 0; b <= oy; b++)
                    for (int a = 0; a <= ox; a++) {
                        const int64_t s = c.slot_of(ci + a, cj + b);
                        parent[4 * l + cnt++] = s < 0 ? -1 : cm[s];
                    }
                for (; cnt < 4; cnt++) parent[4 * l + cnt] = -1;
            }
        }
    }
    return MG_OK;
}

int mg_level_coeffs(mg_handle h, int level, double* h_lambda, double* h_c, void* stream) {
    if (!h || level < 0 || level >= h->L) return MG_EINVAL;
    if (!h->have_coeffs) return MG_ENOTREADY;
    cudaStream_t s = (cudaStream_t)stream;
    const HostLevel& lv = h->hh.lev[level];
    std::vector<double> tmp((size_t)lv.nslots());
    for (int k = 0; k < 2; k++) {
        double* out = k ? h_c : h_lambda;
        if (!out) continue;
        CU(cudaMemcpyAsync(tmp.data(), k ? h->buf[level].c : h->buf[level].lam, tmp.size() * sizeof(double), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        for (int64_t q = 0; q < lv.n; q++) out[q] = tmp[lv.canon2slot[q]];
    }
    return MG_OK;
}

int mg_level_xi(mg_handle h, int level, double* h_xi, void* stream) {
    if (!h || level < 0 || level >= h->L || !h_xi) return MG_EINVAL;
    if (!h->have_coeffs) return MG_ENOTREADY;
    cudaStream_t s = (cudaStream_t)stream;
    const HostLevel& lv = h->hh.lev[level];
    if (!h->three_field) { for (int64_t q = 0; q < lv.n; q++) h_xi[q] = 1.0; return MG_OK; }
    std::vector<double> tmp((size_t)lv.nslots());
    CU(cudaMemcpyAsync(tmp.data(), h->buf[level].xi, tmp.size() * sizeof(double), cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    for (int64_t q = 0; q < lv.n; q++) h_xi[q] = tmp[lv.canon2slot[q]];
    return MG_OK;
}

// ============================================================================ single steps (parity tests)
#define CHECK_LEVEL(cond) do { if (!h || !(cond)) return MG_EINVAL; if (h->host_only) return MG_ECUDA; if (!h->have_coeffs) return MG_ENOTREADY; \
        { int rc__ = check_coeffs(h, (cudaStream_t)stream); if (rc__) return rc__; } } while (0)

int mg_apply(mg_handle h, int level, const double* d_x, double* d_y, void* stream) {
    CHECK_LEVEL(level >= 0 && level < h->L && d_x && d_y);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    const int64_t n = h->hh.lev[level].n;
    launch_gather(L, d_x, h->buf[level].canon2slot, h->buf[level].x, n, 0);
    launch_apply(L, h->lev[level], vec(h->buf[level].x), vec(nullptr), vec(h->buf[level].d), 0);
    launch_scatter(L, h->buf[level].d, h->buf[level].canon2slot, d_y, n, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

int mg_smooth(mg_handle h, int level, double* d_x, const double* d_b, int sweeps, void* stream) {
    CHECK_LEVEL(level >= 0 && level < h->L && d_x && d_b && sweeps >= 0);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    const int64_t n = h->hh.lev[level].n;
    launch_gather(L, d_x, h->buf[level].canon2slot, h->buf[level].x, n, 0);
    launch_gather(L, d_b, h->buf[level].canon2slot, h->buf[level].tb, n, 0);
    CU(cudaEventRecord(h->ev[4], L.stream));
    VecRef fin = enqueue_smooth(L, h->lev[level], vec(h->buf[level].x), vec(h->buf[level].x2), vec(h->buf[level].tb), sweeps, false);
    CU(cudaEventRecord(h->ev[5], L.stream));
    h->step_timed = true;
    launch_scatter(L, fin.base, h->buf[level].canon2slot, d_x, n, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

int mg_smooth_restrict(mg_handle h, int level, double* d_x, const double* d_b, int sweeps, double* d_coarse, void* stream) {
    CHECK_LEVEL(level >= 0 && level + 1 < h->L && d_x && d_b && d_coarse && sweeps >= 1);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    const int64_t n = h->hh.lev[level].n;
    launch_gather(L, d_x, h->buf[level].canon2slot, h->buf[level].x, n, 0);
    launch_gather(L, d_b, h->buf[level].canon2slot, h->buf[level].tb, n, 0);
    CU(cudaEventRecord(h->ev[4], L.stream));
    VecRef fin = enqueue_smooth(L, h->lev[level], vec(h->buf[level].x), vec(h->buf[level].x2), vec(h->buf[level].tb), sweeps, false,
                                &h->lev[level + 1], h->buf[level + 1].b);
    CU(cudaEventRecord(h->ev[5], L.stream));
    h->step_timed = true;
    launch_scatter(L, fin.base, h->buf[level].canon2slot, d_x, n, 0);
    launch_scatter(L, h->buf[level + 1].b, h->buf[level + 1].canon2slot, d_coarse, h->hh.lev[level + 1].n, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

int mg_restrict(mg_handle h, int level, const double* d_fine, double* d_coarse, void* stream) {
    CHECK_LEVEL(level >= 0 && level + 1 < h->L && d_fine && d_coarse);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    launch_gather(L, d_fine, h->buf[level].canon2slot, h->buf[level].d, h->hh.lev[level].n, 0);
    launch_restrict(L, h->lev[level], h->lev[level + 1], h->buf[level].d, h->buf[level + 1].b);
    launch_scatter(L, h->buf[level + 1].b, h->buf[level + 1].canon2slot, d_coarse, h->hh.lev[level + 1].n, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

int mg_prolong_correct(mg_handle h, int level, const double* d_coarse_e, double* d_x_fine, void* stream) {
    CHECK_LEVEL(level >= 0 && level + 1 < h->L && d_coarse_e && d_x_fine);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    launch_gather(L, d_coarse_e, h->buf[level + 1].canon2slot, h->buf[level + 1].x, h->hh.lev[level + 1].n, 0);
    launch_gather(L, d_x_fine, h->buf[level].canon2slot, h->buf[level].x, h->hh.lev[level].n, 0);
    launch_prolong_correct(L, h->lev[level], h->lev[level + 1], h->buf[level + 1].x, h->buf[level].d, vec(h->buf[level].x));
    launch_scatter(L, h->buf[level].x, h->buf[level].canon2slot, d_x_fine, h->hh.lev[level].n, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

int mg_coarse_solve(mg_handle h, const double* d_b, double* d_x, void* stream) {
    CHECK_LEVEL(d_b && d_x);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    const int l = h->L - 1;
    launch_gather(L, d_b, h->buf[l].canon2slot, h->buf[l].tb, h->nL, 0);
    launch_coarse_solve(L, h->Ainv, h->cslot, h->nL, vec(h->buf[l].tb), vec(h->buf[l].x));
    launch_scatter(L, h->buf[l].x, h->buf[l].canon2slot, d_x, h->nL, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

int mg_vcycle(mg_handle h, int level, double* d_x, const double* d_b, void* stream) {
    CHECK_LEVEL(level >= 0 && level < h->L && d_x && d_b);
    Launch L = LZ1(h, (cudaStream_t)stream);      // plane 0
    const int64_t n = h->hh.lev[level].n;
    // level buffers x/b of `level` are free here: the recursion only uses those of the coarser levels
    launch_gather(L, d_x, h->buf[level].canon2slot, h->buf[level].x, n, 0);
    launch_gather(L, d_b, h->buf[level].canon2slot, h->buf[level].tb, n, 0);
    enqueue_cycle(h, L, level, vec(h->buf[level].x), vec(h->buf[level].tb), false);
    CU(h->tail_err);
    launch_scatter(L, h->buf[level].x, h->buf[level].canon2slot, d_x, n, 0);
    CU(cudaGetLastError());
    return MG_OK;
}

}  // extern "C"
