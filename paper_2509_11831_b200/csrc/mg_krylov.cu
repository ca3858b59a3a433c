// fGMRES(m) vector kernels (rules K1-K5; Saad's flexible GMRES).  The paper drives
// GMRES from the host through a reverse-communication interface; here the Hessenberg
// column, Givens rotations, least-squares right-hand side and the stop test (Eq. 23) stay
// on the device in GmresState; every kernel reads the running column index j from it, so one captured
// graph serves all iterations.
//
// Orthogonalisation: classical Gram-Schmidt applied twice (CGS2).  Same Krylov iterates as the oracle's modified
// Gram-Schmidt (also applied twice) up to rounding.  For restart lengths m <= 32 the two projections take
// THREE passes over the basis (k_multidot_tma, k_update_dot_tma, k_final_v: see the block comment further down),
// the first two staged through shared memory by TMA bulk copies, the third skipped in the steps whose measured
// orthogonality defect is already below REORTH_TOL (k_scale_v instead); longer restarts use the plain four-pass
// form (k_multidot, k_update_w twice, k_givens, k_next_v).  Grid reductions: per-block partials +
// last-block-done ticket, summed in a fixed order (deterministic run to run).
#include <algorithm>
#include <cstdlib>

#include "mg_device.h"

namespace mgb {

namespace {

constexpr int CH = 8;   // basis vectors per register chunk in the multi-dot
constexpr int64_t PARTIAL_PLANE = (int64_t)RED_BLOCKS_MAX * (MAX_M + 2);   // doubles of block partials per plane

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Block-level sum; result valid in thread 0.
__device__ __forceinline__ double block_sum(double v, double* sm) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = (threadIdx.x < (blockDim.x >> 5)) ? sm[threadIdx.x] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

// true in every thread of the block that arrived last
__device__ __forceinline__ bool last_block(GmresState* st) {
    __shared__ int is_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const int t = atomicAdd(&st->ticket, 1);
        is_last = (t == (int)gridDim.x - 1);
        if (is_last) st->ticket = 0;
    }
    __syncthreads();
    if (is_last) __threadfence();
    return is_last;
}

__global__ void __launch_bounds__(RED_THREADS) k_norm2(const double* __restrict__ v, int64_t n, GmresState* st,
                                                      double* __restrict__ partial, int which) {
    v += blockIdx.y * n; st += blockIdx.y; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    __shared__ double sm[32];
    double acc = 0.0;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const double a = v[k];
        acc += a * a;
    }
    acc = block_sum(acc, sm);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
    if (last_block(st)) {
        double s = 0.0;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) s += ((volatile double*)partial)[b];
        s = block_sum(s, sm);
        if (threadIdx.x == 0) {
            if (which == 0) st->bn = sqrt(s); else st->beta = sqrt(s);
        }
    }
}

// K1/K2/K5: relres = beta / bn decides converged / restart; v_0 = r / beta; g = (beta, 0, ...).
__global__ void k_start_cycle(GmresState* st, const double* __restrict__ r, double* __restrict__ V0, int64_t n) {
    st += blockIdx.y; r += blockIdx.y * n; V0 += (int64_t)blockIdx.y * (st->m + 1) * n;   // plane = blockIdx.y
    const double beta = st->beta, bn = st->bn;
    const double relres = (bn > 0.0) ? beta / bn : 0.0;
    const bool conv = (bn == 0.0) || (relres < st->rtol);
    const bool capped = st->iters >= st->max_iters;
    const bool broke = st->status == 3;
    __syncthreads();
    if (!conv && !capped && !broke) {
        const double inv = 1.0 / beta;
        for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) V0[k] = r[k] * inv;
    }
    // the header is rewritten by one thread after every block has read it
    if (last_block(st) && threadIdx.x == 0) {
        st->relres = relres;
        if (conv || broke || capped) st->j = 0;                         // no cycle runs: a later k_update_x adds nothing
        if (bn == 0.0) { st->status = 4; st->cycle_end = 1; }           // zero right-hand side: x = 0 (K1)
        else if (conv) { st->status = 1; st->cycle_end = 1; }
        else if (broke) { st->cycle_end = 1; }
        else if (capped) { st->status = 2; st->cycle_end = 1; }
        else { st->status = 0; st->cycle_end = 0; st->j = 0; st->g[0] = beta; }
    }
}

// red[i] = (w, v_i), i = 0..j.  One pass over w per chunk of CH basis vectors.
__global__ void __launch_bounds__(RED_THREADS) k_multidot(const double* __restrict__ w, const double* __restrict__ V, int64_t stride,
                                                         int64_t n, GmresState* st, double* __restrict__ partial) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    __shared__ double sm[32];
    if (st->cycle_end) return;
    const int nv = st->j + 1;
    for (int i0 = 0; i0 < nv; i0 += CH) {
        double acc[CH];
#pragma unroll
        for (int c = 0; c < CH; c++) acc[c] = 0.0;
        const int nc = min(CH, nv - i0);
        for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
            const double wk = w[k];
#pragma unroll
            for (int c = 0; c < CH; c++)
                if (c < nc) acc[c] += wk * V[(int64_t)(i0 + c) * stride + k];
        }
#pragma unroll
        for (int c = 0; c < CH; c++) {
            const double s = block_sum(acc[c], sm);
            if (threadIdx.x == 0 && c < nc) partial[(size_t)blockIdx.x * (MAX_M + 2) + i0 + c] = s;
        }
    }
    if (last_block(st)) {
        for (int i = threadIdx.x; i < nv; i += blockDim.x) {
            double s = 0.0;
            for (int b = 0; b < (int)gridDim.x; b++) s += ((volatile double*)partial)[(size_t)b * (MAX_M + 2) + i];
            st->red[i] = s;
        }
    }
}

// w -= sum_i red[i] v_i ; hcol (+)= red ; hcol[j+1] = ||w||.
__global__ void __launch_bounds__(RED_THREADS) k_update_w(double* __restrict__ w, const double* __restrict__ V, int64_t stride, int64_t n,
                                                         GmresState* st, double* __restrict__ partial, int pass) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    __shared__ double sm[32];
    __shared__ double hh[MAX_M + 1];
    if (st->cycle_end) return;
    const int nv = st->j + 1;
    for (int i = threadIdx.x; i < nv; i += blockDim.x) hh[i] = st->red[i];
    __syncthreads();
    double acc = 0.0;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        double s = w[k];
#pragma unroll 4
        for (int i = 0; i < nv; i++) s -= hh[i] * V[(int64_t)i * stride + k];
        w[k] = s;
        acc += s * s;
    }
    acc = block_sum(acc, sm);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * (MAX_M + 2) + MAX_M + 1] = acc;
    if (last_block(st)) {
        double s = 0.0;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) s += ((volatile double*)partial)[(size_t)b * (MAX_M + 2) + MAX_M + 1];
        s = block_sum(s, sm);
        for (int i = threadIdx.x; i < nv; i += blockDim.x) st->hcol[i] = (pass == 0) ? hh[i] : st->hcol[i] + hh[i];
        if (threadIdx.x == 0) st->hcol[nv] = sqrt(s);
    }
}

// K2/K3: rotate the new Hessenberg column (st->hcol[0..j+1]), update g, count the iteration, evaluate the
// stop test.  Serial, one thread.
__device__ void givens_step(GmresState* st) {
    const int j = st->j, m = st->m;
    double* H = st->H;
    for (int i = 0; i <= j + 1; i++) H[i * MAX_M + j] = st->hcol[i];
    const double hn = st->hcol[j + 1];
    for (int i = 0; i < j; i++) {
        const double a = H[i * MAX_M + j], b = H[(i + 1) * MAX_M + j];
        H[i * MAX_M + j] = st->cs[i] * a + st->sn[i] * b;
        H[(i + 1) * MAX_M + j] = -st->sn[i] * a + st->cs[i] * b;
    }
    const double rho = hypot(H[j * MAX_M + j], hn);
    st->cs[j] = H[j * MAX_M + j] / rho;
    st->sn[j] = hn / rho;
    H[j * MAX_M + j] = rho;
    H[(j + 1) * MAX_M + j] = 0.0;
    st->g[j + 1] = -st->sn[j] * st->g[j];
    st->g[j] = st->cs[j] * st->g[j];
    st->iters += 1;
    const double rel = fabs(st->g[j + 1]) / st->bn;
    if (st->iters <= 512) st->hist[st->iters - 1] = rel;
    st->hn = hn;
    st->inv_hn = hn > 0.0 ? 1.0 / hn : 0.0;
    st->j = j + 1;
    if (rel < st->rtol) st->cycle_end = 1;                              // K3 (confirmed by the true residual, K5)
    else if (hn == 0.0) { st->status = 3; st->cycle_end = 1; }          // breakdown
    else if (j + 1 >= m || st->iters >= st->max_iters) st->cycle_end = 1;
}

__global__ void k_givens(GmresState* st) {
    st += blockIdx.y;   // plane = blockIdx.y
    if (threadIdx.x != 0 || st->cycle_end) return;
    givens_step(st);
}

// ---------------------------------------------------------------------------- fused CGS2 (m <= FUSED_NV)
// Three passes over the basis per Arnoldi step instead of four:
//   pass 1  k_multidot      h1 = V^T w
//   pass 2  k_update_dot    w' = w - V h1 (written), h2 = V^T w', ||w'||^2 — V is read ONCE: the values used
//                           for the update stay in registers for the second set of dot products; the last
//                           block then forms h = h1 + h2, h_{j+1,j} = sqrt(||w'||^2 - sum h2^2) (exact for
//                           orthonormal V; h2 = O(eps) after the first projection so nothing cancels) and runs
//                           the Givens step, so no separate norm pass and no separate Givens launch
//   pass 3  k_final_v       v_{j+1} = (w' - V h2) / h_{j+1,j}, written straight into the basis; where
//                           ||h2|| <= REORTH_TOL ||w'|| (decided in pass 2's last block) the step keeps h = h1,
//                           h_{j+1,j} = ||w'|| and k_scale_v writes v_{j+1} = w' / ||w'|| without reading the basis
// Traffic at column j: 8(j+2) + (16 + 8(j+1)) + (16 + 8(j+1)) = 24 j + 64 B/pt against 32 j + 96.
constexpr int FUSED_NV = 32;
constexpr double REORTH_TOL = 1e-13;   // second update skipped when ||V^T w'|| <= REORTH_TOL ||w'|| (G23)
constexpr int UD_THREADS = 128;
// register-staged variant: 254 registers x 128 threads, two blocks per SM, one wave

// One grid-stride sweep with NV basis values x EPT elements held in registers per thread.
template <int NV, int EPT>
__device__ __forceinline__ void update_dot_body(double* __restrict__ w, const double* __restrict__ V, int64_t stride, int64_t n,
                                                int nv, const double* hh, double (&acc)[FUSED_NV], double& accn) {
    const int64_t G = (int64_t)gridDim.x * blockDim.x;
    for (int64_t k0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k0 < n; k0 += G * EPT) {
        double v[EPT][NV], s[EPT];
#pragma unroll
        for (int e = 0; e < EPT; e++) {
            const int64_t k = k0 + e * G;
            const bool ok = k < n;
            s[e] = ok ? w[k] : 0.0;
#pragma unroll
            for (int c = 0; c < NV; c++) v[e][c] = (ok && c < nv) ? V[(int64_t)c * stride + k] : 0.0;
        }
#pragma unroll
        for (int e = 0; e < EPT; e++) {
            const int64_t k = k0 + e * G;
#pragma unroll
            for (int c = 0; c < NV; c++) s[e] -= hh[c] * v[e][c];
            if (k < n) w[k] = s[e];
            accn += s[e] * s[e];
#pragma unroll
            for (int c = 0; c < NV; c++) acc[c] += s[e] * v[e][c];
        }
    }
}

// Block + grid reduction of the second projection and the Givens step in the last block to arrive.
template <int THREADS>
__device__ __forceinline__ void ud_finish(double (&acc)[FUSED_NV], double accn, int nv, const double* hh, GmresState* st,
                                          double* __restrict__ partial) {
    __shared__ double red[THREADS / 32][FUSED_NV + 1];
    __shared__ double tot[FUSED_NV + 1];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) {
        const double r = warp_sum(acc[c]);
        if (lane == 0) red[warp][c] = r;
    }
    accn = warp_sum(accn);
    if (lane == 0) red[warp][FUSED_NV] = accn;
    __syncthreads();
    if (threadIdx.x <= FUSED_NV) {
        double r = 0.0;
        for (int q = 0; q < THREADS / 32; q++) r += red[q][threadIdx.x];
        partial[(size_t)blockIdx.x * (MAX_M + 2) + threadIdx.x] = r;
    }
    if (last_block(st)) {
        if (threadIdx.x <= FUSED_NV) {
            double r = 0.0;
            for (int b = 0; b < (int)gridDim.x; b++) r += ((volatile double*)partial)[(size_t)b * (MAX_M + 2) + threadIdx.x];
            tot[threadIdx.x] = r;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double s2 = 0.0;
            for (int i = 0; i < nv; i++) s2 += tot[i] * tot[i];
            // h2 = V^T w' IS the orthogonality defect of w' against the basis: when it is below REORTH_TOL
            // relative to ||w'|| the second update would change nothing above that level and is skipped
            // (k_final_v then only normalises: 16 B/pt instead of 8(j+3)).
            const bool skip = st->reorth_tol > 0.0 && s2 <= st->reorth_tol * st->reorth_tol * tot[FUSED_NV];
            for (int i = 0; i < nv; i++) {
                st->hcol[i] = skip ? hh[i] : hh[i] + tot[i];     // h_ij = first (+ second) projection
                st->red[i] = tot[i];                             // h2, consumed by k_final_v
            }
            const double hn2 = skip ? tot[FUSED_NV] : tot[FUSED_NV] - s2;
            st->hcol[nv] = hn2 > 0.0 ? sqrt(hn2) : 0.0;
            st->skip2 = skip ? 1 : 0;
            if (!skip) st->nreorth += 1;
            if (st->iters < 512) st->orth[st->iters] = tot[FUSED_NV] > 0.0 ? sqrt(s2 / tot[FUSED_NV]) : 0.0;
            givens_step(st);
        }
    }
}

__global__ void __launch_bounds__(UD_THREADS) k_update_dot(double* __restrict__ w, const double* __restrict__ V, int64_t stride,
                                                            int64_t n, GmresState* st, double* __restrict__ partial) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    __shared__ double hh[FUSED_NV];
    if (st->cycle_end) return;
    const int nv = st->j + 1;
    if (threadIdx.x < FUSED_NV) hh[threadIdx.x] = threadIdx.x < nv ? st->red[threadIdx.x] : 0.0;
    __syncthreads();
    double acc[FUSED_NV], accn = 0.0;
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) acc[c] = 0.0;
    if (nv <= 8) update_dot_body<8, 4>(w, V, stride, n, nv, hh, acc, accn);
    else if (nv <= 16) update_dot_body<16, 2>(w, V, stride, n, nv, hh, acc, accn);
    else update_dot_body<32, 1>(w, V, stride, n, nv, hh, acc, accn);
    ud_finish<UD_THREADS>(acc, accn, nv, hh, st, partial);
}

// ---- the same pass with the basis chunk staged in shared memory by TMA bulk copies (cp.async.bulk +
// mbarrier, three stages): the bytes in flight no longer depend on registers (two 72 KB stages per SM are
// always outstanding), and both uses of the basis values (update, second projection) read shared memory.
constexpr int UDT_THREADS = 256, UDT_STAGES = 3;
constexpr int UDT_STAGE_DOUBLES = (8 + 1) * UDT_THREADS * 4;          // largest (NV + 1) * K over the three tilings
constexpr size_t UDT_SMEM = (size_t)UDT_STAGES * UDT_STAGE_DOUBLES * sizeof(double) + 64;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!done);
}

// UPDATE = false: pass 1 only (acc = V^T w; w untouched, hh unused).
template <int NV, int EPT, bool UPDATE = true>
__device__ __forceinline__ void update_dot_tma_body(double* __restrict__ w, const double* __restrict__ V, int64_t stride, int64_t n,
                                                    int nv, const double* hh, double (&acc)[FUSED_NV], double& accn, double* stage0,
                                                    uint64_t* bars) {
    constexpr int K = UDT_THREADS * EPT;                    // elements per chunk
    static_assert((NV + 1) * K <= UDT_STAGE_DOUBLES, "stage too small");
    const int64_t nchunks = n / K;                          // n is a multiple of the tile size 2048
    const int tid = threadIdx.x;
    auto issue = [&](int64_t i) {                           // chunk i of this CTA -> stage i % STAGES
        const int64_t ci = (int64_t)blockIdx.x + i * gridDim.x;
        if (ci >= nchunks || tid != 0) return;
        const int sg = (int)(i % UDT_STAGES);
        double* sv = stage0 + (size_t)sg * UDT_STAGE_DOUBLES;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&bars[sg], (uint32_t)((nv + 1) * K * sizeof(double)));
        for (int c = 0; c < nv; c++) bulk_g2s(sv + c * K, V + (int64_t)c * stride + ci * K, K * sizeof(double), &bars[sg]);
        bulk_g2s(sv + NV * K, w + ci * K, K * sizeof(double), &bars[sg]);
    };
    double hr[NV];                                          // the projection coefficients in registers (read once, not once per element)
#pragma unroll
    for (int c = 0; c < NV; c++) hr[c] = (UPDATE && c < nv) ? hh[c] : 0.0;
    for (int i = 0; i < UDT_STAGES; i++) issue(i);           // all stages in flight; a stage is refilled as soon as it is consumed
    for (int64_t i = 0; (int64_t)blockIdx.x + i * gridDim.x < nchunks; i++) {
        const int64_t ci = (int64_t)blockIdx.x + i * gridDim.x;
        const int sg = (int)(i % UDT_STAGES);
        const double* sv = stage0 + (size_t)sg * UDT_STAGE_DOUBLES;
        mbar_wait(&bars[sg], (uint32_t)((i / UDT_STAGES) & 1));
#pragma unroll
        for (int e = 0; e < EPT; e++) {
            const int k = tid + e * UDT_THREADS;
            double s = sv[NV * K + k];
            if (UPDATE) {
#pragma unroll
                for (int c = 0; c < NV; c++)
                    if (c < nv) s -= hr[c] * sv[c * K + k];
                w[ci * K + k] = s;
                accn += s * s;
            }
#pragma unroll
            for (int c = 0; c < NV; c++)
                if (c < nv) acc[c] += s * sv[c * K + k];
        }
        __syncthreads();                                    // everyone is done with this stage: refill it
        issue(i + UDT_STAGES);
    }
}

__global__ void __launch_bounds__(UDT_THREADS, 1) k_update_dot_tma(double* __restrict__ w, const double* __restrict__ V, int64_t stride,
                                                                   int64_t n, GmresState* st, double* __restrict__ partial) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    extern __shared__ __align__(128) unsigned char udt_smem[];
    __shared__ double hh[FUSED_NV];
    if (st->cycle_end) return;
    double* stage0 = reinterpret_cast<double*>(udt_smem);
    uint64_t* bars = reinterpret_cast<uint64_t*>(udt_smem + (size_t)UDT_STAGES * UDT_STAGE_DOUBLES * sizeof(double));
    const int nv = st->j + 1;
    if (threadIdx.x < FUSED_NV) hh[threadIdx.x] = threadIdx.x < nv ? st->red[threadIdx.x] : 0.0;
    if (threadIdx.x == 0) {
        for (int sgi = 0; sgi < UDT_STAGES; sgi++) mbar_init(&bars[sgi], 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    double acc[FUSED_NV], accn = 0.0;
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) acc[c] = 0.0;
    if (nv <= 8) update_dot_tma_body<8, 4>(w, V, stride, n, nv, hh, acc, accn, stage0, bars);
    else if (nv <= 16) update_dot_tma_body<16, 2>(w, V, stride, n, nv, hh, acc, accn, stage0, bars);
    else update_dot_tma_body<32, 1>(w, V, stride, n, nv, hh, acc, accn, stage0, bars);
    ud_finish<UDT_THREADS>(acc, accn, nv, hh, st, partial);
}

template <int NV, int EPT>
__device__ __forceinline__ void multidot_body(const double* __restrict__ w, const double* __restrict__ V, int64_t stride, int64_t n,
                                              int nv, double (&acc)[FUSED_NV]) {
    const int64_t G = (int64_t)gridDim.x * blockDim.x;
    for (int64_t k0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k0 < n; k0 += G * EPT) {
        double v[EPT][NV], wk[EPT];
#pragma unroll
        for (int e = 0; e < EPT; e++) {
            const int64_t k = k0 + e * G;
            const bool ok = k < n;
            wk[e] = ok ? w[k] : 0.0;
#pragma unroll
            for (int c = 0; c < NV; c++) v[e][c] = (ok && c < nv) ? V[(int64_t)c * stride + k] : 0.0;
        }
#pragma unroll
        for (int e = 0; e < EPT; e++)
#pragma unroll
            for (int c = 0; c < NV; c++) acc[c] += wk[e] * v[e][c];
    }
}

constexpr int MD_THREADS = 256;
__global__ void __launch_bounds__(MD_THREADS, 2) k_multidot_t(const double* __restrict__ w, const double* __restrict__ V, int64_t stride,
                                                              int64_t n, GmresState* st, double* __restrict__ partial) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    __shared__ double red[MD_THREADS / 32][FUSED_NV];
    if (st->cycle_end) return;
    const int nv = st->j + 1;
    double acc[FUSED_NV];
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) acc[c] = 0.0;
    if (nv <= 8) multidot_body<8, 4>(w, V, stride, n, nv, acc);
    else if (nv <= 16) multidot_body<16, 2>(w, V, stride, n, nv, acc);
    else multidot_body<32, 1>(w, V, stride, n, nv, acc);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) {
        const double r = warp_sum(acc[c]);
        if (lane == 0) red[warp][c] = r;
    }
    __syncthreads();
    if (threadIdx.x < FUSED_NV) {
        double r = 0.0;
        for (int q = 0; q < MD_THREADS / 32; q++) r += red[q][threadIdx.x];
        partial[(size_t)blockIdx.x * (MAX_M + 2) + threadIdx.x] = r;
    }
    if (last_block(st)) {
        if ((int)threadIdx.x < nv) {
            double r = 0.0;
            for (int b = 0; b < (int)gridDim.x; b++) r += ((volatile double*)partial)[(size_t)b * (MAX_M + 2) + threadIdx.x];
            st->red[threadIdx.x] = r;
        }
    }
}

// Pass 1 through the same TMA pipeline.
__global__ void __launch_bounds__(UDT_THREADS, 1) k_multidot_tma(double* __restrict__ w, const double* __restrict__ V, int64_t stride,
                                                                 int64_t n, GmresState* st, double* __restrict__ partial) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride; partial += blockIdx.y * PARTIAL_PLANE;   // plane = blockIdx.y
    extern __shared__ __align__(128) unsigned char udt_smem[];
    __shared__ double red[UDT_THREADS / 32][FUSED_NV];
    if (st->cycle_end) return;
    double* stage0 = reinterpret_cast<double*>(udt_smem);
    uint64_t* bars = reinterpret_cast<uint64_t*>(udt_smem + (size_t)UDT_STAGES * UDT_STAGE_DOUBLES * sizeof(double));
    const int nv = st->j + 1;
    if (threadIdx.x == 0) {
        for (int sgi = 0; sgi < UDT_STAGES; sgi++) mbar_init(&bars[sgi], 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    double acc[FUSED_NV], accn = 0.0;
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) acc[c] = 0.0;
    if (nv <= 8) update_dot_tma_body<8, 4, false>(w, V, stride, n, nv, nullptr, acc, accn, stage0, bars);
    else if (nv <= 16) update_dot_tma_body<16, 2, false>(w, V, stride, n, nv, nullptr, acc, accn, stage0, bars);
    else update_dot_tma_body<32, 1, false>(w, V, stride, n, nv, nullptr, acc, accn, stage0, bars);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int c = 0; c < FUSED_NV; c++) {
        const double r = warp_sum(acc[c]);
        if (lane == 0) red[warp][c] = r;
    }
    __syncthreads();
    if (threadIdx.x < FUSED_NV) {
        double r = 0.0;
        for (int q = 0; q < UDT_THREADS / 32; q++) r += red[q][threadIdx.x];
        partial[(size_t)blockIdx.x * (MAX_M + 2) + threadIdx.x] = r;
    }
    if (last_block(st)) {
        if ((int)threadIdx.x < nv) {
            double r = 0.0;
            for (int b = 0; b < (int)gridDim.x; b++) r += ((volatile double*)partial)[(size_t)b * (MAX_M + 2) + threadIdx.x];
            st->red[threadIdx.x] = r;
        }
    }
}

template <int NV, int EPT>
__device__ __forceinline__ void final_v_body(const double* __restrict__ w, const double* __restrict__ V, double* __restrict__ out,
                                             int64_t stride, int64_t n, int nv, const double* hh, double inv) {
    const int64_t G = (int64_t)gridDim.x * blockDim.x;
    for (int64_t k0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k0 < n; k0 += G * EPT) {
        double v[EPT][NV], s[EPT];
#pragma unroll
        for (int e = 0; e < EPT; e++) {
            const int64_t k = k0 + e * G;
            const bool ok = k < n;
            s[e] = ok ? w[k] : 0.0;
#pragma unroll
            for (int c = 0; c < NV; c++) v[e][c] = (ok && c < nv) ? V[(int64_t)c * stride + k] : 0.0;
        }
#pragma unroll
        for (int e = 0; e < EPT; e++) {
            const int64_t k = k0 + e * G;
#pragma unroll
            for (int c = 0; c < NV; c++) s[e] -= hh[c] * v[e][c];
            if (k < n) out[k] = s[e] * inv;
        }
    }
}

// v_{j+1} = (w' - V h2) / h_{j+1,j}; st->j has already been advanced by the Givens step.
__global__ void __launch_bounds__(RED_THREADS) k_final_v(const double* __restrict__ w, double* __restrict__ V, int64_t stride, int64_t n,
                                                        GmresState* st) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride;   // plane = blockIdx.y
    __shared__ double hh[FUSED_NV];
    if (st->cycle_end || st->skip2) return;
    const int nv = st->j;
    double* out = V + (int64_t)nv * stride;
    const double inv = st->inv_hn;
    if (threadIdx.x < FUSED_NV) hh[threadIdx.x] = threadIdx.x < nv ? st->red[threadIdx.x] : 0.0;
    __syncthreads();
    if (nv <= 8) final_v_body<8, 4>(w, V, out, stride, n, nv, hh, inv);
    else if (nv <= 16) final_v_body<16, 2>(w, V, out, stride, n, nv, hh, inv);
    else final_v_body<32, 1>(w, V, out, stride, n, nv, hh, inv);
}

// The step needs no second update (skip2, see ud_finish): v_{j+1} = w' / h_{j+1,j}.  n is a multiple of the tile size.
constexpr int SV_THREADS = 256, SV_UNROLL = 4;
__global__ void __launch_bounds__(SV_THREADS) k_scale_v(const double* __restrict__ w, double* __restrict__ V, int64_t stride, int64_t n,
                                                        GmresState* st) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride;   // plane = blockIdx.y
    if (st->cycle_end || !st->skip2) return;
    const double inv = st->inv_hn;
    const double2* __restrict__ w2 = reinterpret_cast<const double2*>(w);
    double2* __restrict__ o2 = reinterpret_cast<double2*>(V + (int64_t)st->j * stride);
    const int64_t n2 = n >> 1, G = (int64_t)gridDim.x * SV_THREADS;
    for (int64_t k0 = (int64_t)blockIdx.x * SV_THREADS + threadIdx.x; k0 < n2; k0 += G * SV_UNROLL) {
        double2 a[SV_UNROLL];
#pragma unroll
        for (int e = 0; e < SV_UNROLL; e++) if (k0 + e * G < n2) a[e] = w2[k0 + e * G];
#pragma unroll
        for (int e = 0; e < SV_UNROLL; e++) if (k0 + e * G < n2) o2[k0 + e * G] = make_double2(a[e].x * inv, a[e].y * inv);
    }
}

// v_{j+1} = w / h_{j+1,j}
__global__ void k_next_v(const double* __restrict__ w, double* __restrict__ V, int64_t stride, int64_t n, GmresState* st) {
    st += blockIdx.y; w += blockIdx.y * n; V += (int64_t)blockIdx.y * (st->m + 1) * stride;   // plane = blockIdx.y
    if (st->cycle_end) return;
    double* v = V + (int64_t)st->j * stride;
    const double inv = st->inv_hn;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) v[k] = w[k] * inv;
}

// K4: back-substitute R y = g (tiny; redone by every block), x += sum_i y_i z_i.
__global__ void __launch_bounds__(256) k_update_x(double* __restrict__ x, const double* __restrict__ Z, int64_t stride, int64_t n, GmresState* st) {
    st += blockIdx.y; x += blockIdx.y * n; Z += (int64_t)blockIdx.y * (st->m + 1) * stride;   // plane = blockIdx.y
    __shared__ double y[MAX_M];
    const int nv = st->j;
    if (threadIdx.x == 0) {
        for (int i = nv - 1; i >= 0; i--) {
            double s = st->g[i];
            for (int k = i + 1; k < nv; k++) s -= st->H[i * MAX_M + k] * y[k];
            y[i] = s / st->H[i * MAX_M + i];
        }
    }
    __syncthreads();
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        double s = x[k];
#pragma unroll 4
        for (int i = 0; i < nv; i++) s += y[i] * Z[(int64_t)i * stride + k];
        x[k] = s;
    }
}

__global__ void k_init_state(GmresState* st, int m, int max_iters, double rtol, double reorth_tol) {
    st += blockIdx.y;   // plane = blockIdx.y
    if (threadIdx.x != 0) return;
    st->nreorth = 0; st->skip2 = 0; st->reorth_tol = reorth_tol;
    st->j = 0; st->iters = 0; st->status = 0; st->cycle_end = 0; st->m = m; st->max_iters = max_iters;
    st->ticket = 0; st->rtol = rtol; st->bn = 0.0; st->beta = 0.0; st->relres = 0.0; st->hn = 0.0; st->inv_hn = 0.0;
}

// K1: a plane whose right-hand side is zero (status 4) has the solution x = 0
__global__ void k_zero_rhs_planes(double* __restrict__ x, int64_t n, const GmresState* st) {
    st += blockIdx.y;
    if (st->status != 4) return;
    x += blockIdx.y * n;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) x[k] = 0.0;
}

inline void count(const Launch& L, int k = 1) { if (L.counter) *L.counter += k; }
// CTAs per plane of the TMA-staged passes: one per SM, fewer for short vectors so that every CTA streams at least four
// chunks through its pipeline.  A function of the vector length only — not of the number of planes — because the
// block count fixes the summation tree: a batched handle must reduce exactly like a single-plane one.
inline int tma_blocks(int64_t n, int sms) {
    static const int div = getenv("MG_B200_TMA_DIV") ? atoi(getenv("MG_B200_TMA_DIV")) : 4;
    return (int)std::max<int64_t>(1, std::min<int64_t>(sms, n / (UDT_THREADS * 4) / div));
}

}  // namespace

void launch_zero_rhs_planes(const Launch& L, double* x, int64_t n, const GmresState* st) {
    k_zero_rhs_planes<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(x, n, st); count(L);
}
void launch_norm2(const Launch& L, const double* v, int64_t n, GmresState* st, double* partial, int which) {
    k_norm2<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(v, n, st, partial, which); count(L);
}
void launch_start_cycle(const Launch& L, GmresState* st, const double* r, double* V0, int64_t n) {
    k_start_cycle<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, r, V0, n); count(L);
}
void launch_multidot(const Launch& L, const double* w, const double* V, int64_t stride, int64_t n, GmresState* st, double* partial, int m) {
    static const bool no_tma = getenv("MG_B200_NO_TMA") != nullptr;
    if (!no_tma) ensure_dyn_smem((const void*)k_multidot_tma, UDT_SMEM);
    const int sms = dev_info().sms;
    if (m <= FUSED_NV && !no_tma && n % (UDT_THREADS * 4) == 0)
        k_multidot_tma<<<dim3(tma_blocks(n, sms), L.planes), UDT_THREADS, UDT_SMEM, L.stream>>>(const_cast<double*>(w), V, stride, n, st, partial);
    else if (m <= FUSED_NV) k_multidot_t<<<dim3(sms * 2, L.planes), MD_THREADS, 0, L.stream>>>(w, V, stride, n, st, partial);
    else k_multidot<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(w, V, stride, n, st, partial);
    count(L);
}
void launch_update_w(const Launch& L, double* w, const double* V, int64_t stride, int64_t n, GmresState* st, double* partial, int pass) {
    k_update_w<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(w, V, stride, n, st, partial, pass); count(L);
}
void launch_update_dot(const Launch& L, double* w, const double* V, int64_t stride, int64_t n, GmresState* st, double* partial) {
    static const bool no_tma = getenv("MG_B200_NO_TMA") != nullptr;
    if (!no_tma) ensure_dyn_smem((const void*)k_update_dot_tma, UDT_SMEM);
    const int sms = dev_info().sms;
    if (!no_tma && n % (UDT_THREADS * 4) == 0) k_update_dot_tma<<<dim3(tma_blocks(n, sms), L.planes), UDT_THREADS, UDT_SMEM, L.stream>>>(w, V, stride, n, st, partial);
    else k_update_dot<<<dim3(sms * 2, L.planes), UD_THREADS, 0, L.stream>>>(w, V, stride, n, st, partial);
    count(L);
}
void launch_final_v(const Launch& L, const double* w, double* V, int64_t stride, int64_t n, GmresState* st) {
    k_final_v<<<dim3(dev_info().sms * 2, L.planes), RED_THREADS, 0, L.stream>>>(w, V, stride, n, st); count(L);
    k_scale_v<<<dim3(dev_info().sms * 8, L.planes), SV_THREADS, 0, L.stream>>>(w, V, stride, n, st); count(L);
}
void launch_givens(const Launch& L, GmresState* st) { k_givens<<<dim3(1, L.planes), 32, 0, L.stream>>>(st); count(L); }
void launch_next_v(const Launch& L, const double* w, double* V, int64_t stride, int64_t n, GmresState* st) {
    k_next_v<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(w, V, stride, n, st); count(L);
}
void launch_update_x(const Launch& L, double* x, const double* Z, int64_t stride, int64_t n, GmresState* st) {
    k_update_x<<<dim3(red_blocks(), L.planes), 256, 0, L.stream>>>(x, Z, stride, n, st); count(L);
}
void launch_init_state(const Launch& L, GmresState* st, int m, int max_iters, double rtol, bool full_cgs2) {
    static const char* env = getenv("MG_B200_REORTH_TOL");          // experiments only
    const double tol = full_cgs2 ? -1.0 : (env ? atof(env) : REORTH_TOL);
    k_init_state<<<dim3(1, L.planes), 32, 0, L.stream>>>(st, m, max_iters, rtol, tol); count(L);
}

}  // namespace mgb
