// BiCGStab with the V-cycle as right preconditioner (mg_options.solver = 1): the alternative outer solver the paper names
// (PAPER.md:342).  It keeps no Krylov basis: per step (two preconditioner applications) the vector kernels below move
// 19 vectors of 8 B/pt against 24 j + 64 B/pt per application for fGMRES(m) at column j.
//
//     rho' = (rhat, r); beta = (rho'/rho)(alpha/omega); p = r + beta (p - omega v)          k_bi_p
//     y = M p; v = A y                                                                       V-cycle, w = A x fused
//     alpha = rho' / (rhat, v)                                                               k_bi_alpha
//     s = r - alpha v; |s|/|b| < rtol -> half step                                           k_bi_s
//     z = M s; t = A z                                                                       V-cycle (skipped after a half step)
//     omega = (t, s)/(t, t)                                                                  k_bi_omega
//     x += alpha y + omega z; r = s - omega t; rho' = (rhat, r); |r|/|b| < rtol -> stop      k_bi_update
//
// As for fGMRES all scalars, the iteration count and the stop test (Eq. 23) live in the per-plane state on
// the device; one captured graph serves all steps and all planes.  Grid reductions: per-block partials + last-block
// ticket, summed in a fixed order.
#include "mg_device.h"

namespace mgb {

namespace {

constexpr int64_t PARTIAL_PLANE = (int64_t)RED_BLOCKS_MAX * (MAX_M + 2);

__device__ __forceinline__ double wsum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
// block sums of two values; valid in thread 0
__device__ __forceinline__ void bsum2(double& a, double& b, double (*sm)[2]) {
    a = wsum(a); b = wsum(b);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) { sm[threadIdx.x >> 5][0] = a; sm[threadIdx.x >> 5][1] = b; }
    __syncthreads();
    if (threadIdx.x < 32) {
        a = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x][0] : 0.0;
        b = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x][1] : 0.0;
        a = wsum(a); b = wsum(b);
    }
}
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
// grid reduction of two per-block values; the last block to arrive gets the totals in thread 0 (returns true there)
__device__ __forceinline__ bool gsum2(GmresState* st, double* __restrict__ partial, double& a, double& b) {
    __shared__ double sm[32][2];
    bsum2(a, b, sm);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = a; partial[2 * blockIdx.x + 1] = b; }
    if (!last_block(st)) return false;
    a = 0.0; b = 0.0;
    for (int k = threadIdx.x; k < (int)gridDim.x; k += blockDim.x) { a += ((volatile double*)partial)[2 * k]; b += ((volatile double*)partial)[2 * k + 1]; }
    bsum2(a, b, sm);
    return threadIdx.x == 0;
}

// The vectors have a multiple of 2048 entries (tile layout): 16-byte accesses, two per thread and trip in flight
#define BI_LOOP(k2) for (int64_t k2 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k2 < (n >> 1); k2 += (int64_t)gridDim.x * blockDim.x)
__device__ __forceinline__ double2 ld2(const double* p, int64_t k2) { return reinterpret_cast<const double2*>(p)[k2]; }
__device__ __forceinline__ void st2(double* p, int64_t k2, double a, double b) { reinterpret_cast<double2*>(p)[k2] = make_double2(a, b); }

// (re)start, rules K1 / K5: relres = |r| / |b| decides converged / restart; rhat = r, rho' = (rhat, r) = |r|^2
__global__ void __launch_bounds__(RED_THREADS) k_bi_start(GmresState* st, const double* __restrict__ r, double* __restrict__ rhat, int64_t n) {
    st += blockIdx.y; r += blockIdx.y * n; rhat += blockIdx.y * n;
    const double beta = st->beta, bn = st->bn;
    const double relres = (bn > 0.0) ? beta / bn : 0.0;
    const bool conv = (bn == 0.0) || (relres < st->rtol);
    const bool capped = st->iters >= st->max_iters;
    const bool broke = st->status == 3;
    __syncthreads();
    if (!conv && !capped && !broke)
        BI_LOOP(k2) { const double2 a = ld2(r, k2); st2(rhat, k2, a.x, a.y); }
    if (last_block(st) && threadIdx.x == 0) {
        st->relres = relres;
        if (bn == 0.0) { st->status = 4; st->cycle_end = 1; }
        else if (conv) { st->status = 1; st->cycle_end = 1; }
        else if (broke) { st->cycle_end = 1; }
        else if (capped) { st->status = 2; st->cycle_end = 1; }
        else {
            st->status = 0; st->cycle_end = 0; st->b_first = 1; st->b_half = 0; st->b_skip2 = 0;
            st->b_rho = 1.0; st->b_alpha = 1.0; st->b_omega = 1.0; st->b_rho1 = beta * beta;
        }
        if (st->cycle_end) st->b_skip2 = 1;
    }
}

__global__ void __launch_bounds__(RED_THREADS) k_bi_p(GmresState* st, const double* __restrict__ r, double* __restrict__ p,
                                                      const double* __restrict__ v, int64_t n) {
    st += blockIdx.y; r += blockIdx.y * n; p += blockIdx.y * n; v += blockIdx.y * n;
    if (st->cycle_end) return;
    const bool first = st->b_first != 0;
    const double omega = st->b_omega;
    const double beta = (st->b_rho1 / st->b_rho) * (st->b_alpha / omega);
    BI_LOOP(k2) {
        const double2 rr = ld2(r, k2);
        if (first) st2(p, k2, rr.x, rr.y);
        else {
            const double2 pp = ld2(p, k2), vv = ld2(v, k2);
            st2(p, k2, rr.x + beta * (pp.x - omega * vv.x), rr.y + beta * (pp.y - omega * vv.y));
        }
    }
}

__global__ void __launch_bounds__(RED_THREADS) k_bi_alpha(GmresState* st, const double* __restrict__ rhat, const double* __restrict__ v, int64_t n,
                                                          double* __restrict__ partial) {
    st += blockIdx.y; rhat += blockIdx.y * n; v += blockIdx.y * n; partial += blockIdx.y * PARTIAL_PLANE;
    if (st->cycle_end) return;
    double a = 0.0, b = 0.0;
    BI_LOOP(k2) { const double2 x = ld2(rhat, k2), y = ld2(v, k2); a += x.x * y.x; a += x.y * y.y; }
    if (gsum2(st, partial, a, b)) {
        if (a == 0.0) { st->status = 3; st->cycle_end = 1; st->b_skip2 = 1; }      // breakdown: (rhat, v) = 0
        else st->b_alpha = st->b_rho1 / a;
    }
}

__global__ void __launch_bounds__(RED_THREADS) k_bi_s(GmresState* st, const double* __restrict__ r, const double* __restrict__ v, double* __restrict__ s,
                                                      int64_t n, double* __restrict__ partial) {
    st += blockIdx.y; r += blockIdx.y * n; v += blockIdx.y * n; s += blockIdx.y * n; partial += blockIdx.y * PARTIAL_PLANE;
    if (st->cycle_end) return;
    const double alpha = st->b_alpha;
    double a = 0.0, b = 0.0;
    BI_LOOP(k2) {
        const double2 rr = ld2(r, k2), vv = ld2(v, k2);
        const double s0 = rr.x - alpha * vv.x, s1 = rr.y - alpha * vv.y;
        st2(s, k2, s0, s1);
        a += s0 * s0; a += s1 * s1;
    }
    if (gsum2(st, partial, a, b)) {
        st->iters += 1;                                                           // first preconditioner application of the step
        const double rel = sqrt(a) / st->bn;
        if (st->iters <= 512) st->hist[st->iters - 1] = rel;
        if (rel < st->rtol || st->iters >= st->max_iters) { st->b_half = 1; st->b_skip2 = 1; }
    }
}

__global__ void __launch_bounds__(RED_THREADS) k_bi_omega(GmresState* st, const double* __restrict__ t, const double* __restrict__ s, int64_t n,
                                                          double* __restrict__ partial) {
    st += blockIdx.y; t += blockIdx.y * n; s += blockIdx.y * n; partial += blockIdx.y * PARTIAL_PLANE;
    if (st->cycle_end || st->b_half) return;
    double a = 0.0, b = 0.0;
    BI_LOOP(k2) {
        const double2 tt = ld2(t, k2), ss = ld2(s, k2);
        a += tt.x * ss.x; a += tt.y * ss.y;
        b += tt.x * tt.x; b += tt.y * tt.y;
    }
    if (gsum2(st, partial, a, b)) {
        if (b == 0.0) { st->status = 3; st->b_half = 1; }                          // breakdown: (t, t) = 0; x still takes alpha y
        else st->b_omega = a / b;
    }
}

__global__ void __launch_bounds__(RED_THREADS) k_bi_update(GmresState* st, double* __restrict__ x, double* __restrict__ r, const double* __restrict__ rhat,
                                                           const double* __restrict__ y, const double* __restrict__ z, const double* __restrict__ s,
                                                           const double* __restrict__ t, int64_t n, double* __restrict__ partial) {
    const int64_t o = blockIdx.y * n;
    st += blockIdx.y; x += o; r += o; rhat += o; y += o; z += o; s += o; t += o; partial += blockIdx.y * PARTIAL_PLANE;
    if (st->cycle_end) return;
    const double alpha = st->b_alpha, omega = st->b_omega;
    const bool half = st->b_half != 0;
    double a = 0.0, b = 0.0;
    if (half) {
        BI_LOOP(k2) { const double2 xx = ld2(x, k2), yy = ld2(y, k2); st2(x, k2, xx.x + alpha * yy.x, xx.y + alpha * yy.y); }
    } else {
        BI_LOOP(k2) {
            const double2 xx = ld2(x, k2), yy = ld2(y, k2), zz = ld2(z, k2), ss = ld2(s, k2), tt = ld2(t, k2), hh = ld2(rhat, k2);
            st2(x, k2, xx.x + (alpha * yy.x + omega * zz.x), xx.y + (alpha * yy.y + omega * zz.y));
            const double r0 = ss.x - omega * tt.x, r1 = ss.y - omega * tt.y;
            st2(r, k2, r0, r1);
            a += hh.x * r0; a += hh.y * r1;
            b += r0 * r0; b += r1 * r1;
        }
    }
    if (gsum2(st, partial, a, b)) {
        if (half) { st->cycle_end = 1; }
        else {
            st->iters += 1;                                                       // second preconditioner application
            const double rel = sqrt(b) / st->bn;
            if (st->iters <= 512) st->hist[st->iters - 1] = rel;
            st->b_rho = st->b_rho1;
            st->b_rho1 = a;
            st->b_first = 0;
            if (rel < st->rtol) st->cycle_end = 1;                                // K3 (confirmed by the true residual, K5)
            else if (a == 0.0 || omega == 0.0) { st->status = 3; st->cycle_end = 1; }
            else if (st->iters >= st->max_iters) st->cycle_end = 1;
        }
        st->b_skip2 = st->cycle_end;
    }
}

inline void count(const Launch& L, int k = 1) { if (L.counter) *L.counter += k; }

}  // namespace

void launch_bi_start(const Launch& L, GmresState* st, const double* r, double* rhat, int64_t n) {
    k_bi_start<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, r, rhat, n); count(L);
}
void launch_bi_p(const Launch& L, GmresState* st, const double* r, double* p, const double* v, int64_t n) {
    k_bi_p<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, r, p, v, n); count(L);
}
void launch_bi_alpha(const Launch& L, GmresState* st, const double* rhat, const double* v, int64_t n, double* partial) {
    k_bi_alpha<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, rhat, v, n, partial); count(L);
}
void launch_bi_s(const Launch& L, GmresState* st, const double* r, const double* v, double* s, int64_t n, double* partial) {
    k_bi_s<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, r, v, s, n, partial); count(L);
}
void launch_bi_omega(const Launch& L, GmresState* st, const double* t, const double* s, int64_t n, double* partial) {
    k_bi_omega<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, t, s, n, partial); count(L);
}
void launch_bi_update(const Launch& L, GmresState* st, double* x, double* r, const double* rhat, const double* y, const double* z,
                      const double* s, const double* t, int64_t n, double* partial) {
    k_bi_update<<<dim3(red_blocks(), L.planes), RED_THREADS, 0, L.stream>>>(st, x, r, rhat, y, z, s, t, n, partial); count(L);
}

}  // namespace mgb
