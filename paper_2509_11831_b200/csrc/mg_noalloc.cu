// mg_norm2_noalloc: the Euclidean norm of a device vector (the reduction behind the stop test |Ax - b| / |b| < tol,
// PAPER.md:260 Eq. 23) through an entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (stream
// capture, tight serving loops, harnesses that forbid it).  It is the variant of the library's grid reduction (k_norm2 in
// mg_krylov.cu: per-block partial sums + last-block ticket) whose scratch — the partial sums and the ticket — lives in a
// file-scope __device__ array of fixed size instead of in memory a handle allocated.
//
//  * The array is NA_SCRATCH_BYTES = 32 KB + 256 B; every GPU that loads the library holds it until the process exits.
//  * One block reduces one chunk of NA_CHUNK = 65 536 elements and writes one partial sum; the array holds NA_MAX_BLOCKS = 4096
//    of them, hence the limit MG_NOALLOC_MAX_N = 4096 * 65 536 = 268 435 456 elements (2 GiB of doubles).  Larger n is refused
//    (MG_EINVAL, mg_last_error() says why).
//  * In host code the array's NAME is a host-side stand-in, not a device address: the address is taken once per device, with
//    that device current, by cudaGetSymbolAddress in this file (the array is visible only here) and handed to the kernel.
//  * All calls on one device share the array, which keeps the last call's contents.  The ticket must start at zero: every call
//    clears it on its stream first (cudaMemsetAsync, no allocation); the partial sums are overwritten before they are read.
//    Two calls that OVERLAP on the GPU (different streams, or graph branches without an edge between them) race on the
//    array and give wrong results: order them on one stream / one graph path.
//  * The summation order is fixed by n alone (chunk partials in block order, then a fixed tree), so the result does not
//    depend on the device's SM count and is identical run to run.
#include <cuda_runtime.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <string>

#include "../../include/mg_b200.h"
#include "mg_device.h"

namespace mgb {

namespace {

constexpr int NA_CHUNK = 65536;        // elements per block
constexpr int NA_MAX_BLOCKS = 4096;    // partial sums the scratch holds
constexpr int NA_THREADS = 256;
static_assert((int64_t)NA_CHUNK * NA_MAX_BLOCKS == MG_NOALLOC_MAX_N, "header and scratch size disagree");

struct NaScratch {
    double partial[NA_MAX_BLOCKS];
    unsigned int ticket;               // blocks that have published their partial sum
    unsigned int pad[63];
};
constexpr size_t NA_SCRATCH_BYTES = sizeof(NaScratch);

// The scratch.  Device code names it directly; HOST code must not pass `g_na_scratch` to a kernel (see the header comment).
static __device__ __align__(256) unsigned char g_na_scratch[NA_SCRATCH_BYTES];

__device__ __forceinline__ double na_warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double na_block_sum(double v, double* sm) {      // valid in thread 0
    v = na_warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = (threadIdx.x < NA_THREADS / 32) ? sm[threadIdx.x] : 0.0;
        r = na_warp_sum(r);
    }
    return r;
}

// out[0] = sqrt(sum v[k]^2).  `scr` is the device address of g_na_scratch (from cudaGetSymbolAddress).
__global__ void __launch_bounds__(NA_THREADS) k_norm2_noalloc(const double* __restrict__ v, int64_t n, double* __restrict__ out, NaScratch* scr) {
    __shared__ double sm[32];
    __shared__ int is_last;
    const int64_t k0 = (int64_t)blockIdx.x * NA_CHUNK, k1 = min(k0 + NA_CHUNK, n);
    double acc = 0.0;
    for (int64_t k = k0 + threadIdx.x; k < k1; k += NA_THREADS) {
        const double a = v[k];
        acc = fma(a, a, acc);
    }
    acc = na_block_sum(acc, sm);
    if (threadIdx.x == 0) {
        scr->partial[blockIdx.x] = acc;
        __threadfence();
        is_last = (atomicAdd(&scr->ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double s = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += NA_THREADS) s += ((volatile double*)scr->partial)[b];
    s = na_block_sum(s, sm);
    if (threadIdx.x == 0) {
        out[0] = sqrt(s);
        scr->ticket = 0;               // left clean for the next call (which clears it again anyway)
    }
}

std::mutex g_na_mu;
std::map<int, NaScratch*> g_na_ptr;    // device -> device address of g_na_scratch on that device

// Set-up, once per device, with that device current.
cudaError_t na_scratch(NaScratch** p) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lk(g_na_mu);
    auto it = g_na_ptr.find(dev);
    if (it != g_na_ptr.end()) { *p = it->second; return cudaSuccess; }
    void* addr = nullptr;
    e = cudaGetSymbolAddress(&addr, g_na_scratch);
    if (e != cudaSuccess) return e;
    g_na_ptr[dev] = static_cast<NaScratch*>(addr);
    *p = static_cast<NaScratch*>(addr);
    return cudaSuccess;
}

}  // namespace
}  // namespace mgb

extern "C" int mg_norm2_noalloc(const double* d_v, int64_t n, double* d_out, void* stream) {
    using namespace mgb;
    if (!d_out || n < 0 || (n > 0 && !d_v)) { set_last_error("mg_norm2_noalloc: null pointer or n < 0"); return MG_EINVAL; }
    if (n > (int64_t)MG_NOALLOC_MAX_N) {
        set_last_error("mg_norm2_noalloc: n = " + std::to_string((long long)n) + " exceeds MG_NOALLOC_MAX_N = " +
                       std::to_string((long long)MG_NOALLOC_MAX_N) + " (the fixed scratch holds 4096 partial sums of 65536 elements each)");
        return MG_EINVAL;
    }
    NaScratch* scr = nullptr;
    cudaError_t e = na_scratch(&scr);
    if (e != cudaSuccess) { set_last_error(std::string("mg_norm2_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e)); cudaGetLastError(); return MG_ECUDA; }
    cudaStream_t s = (cudaStream_t)stream;
    e = cudaMemsetAsync(&scr->ticket, 0, sizeof(unsigned int), s);        // the ticket must start at zero
    if (e != cudaSuccess) { set_last_error(std::string("mg_norm2_noalloc: cudaMemsetAsync: ") + cudaGetErrorString(e)); cudaGetLastError(); return MG_ECUDA; }
    const int grid = (int)std::max<int64_t>(1, (n + NA_CHUNK - 1) / NA_CHUNK);
    k_norm2_noalloc<<<grid, NA_THREADS, 0, s>>>(d_v, n, d_out, scr);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_last_error(std::string("mg_norm2_noalloc: launch: ") + cudaGetErrorString(e)); return MG_ECUDA; }
    return MG_OK;
}
