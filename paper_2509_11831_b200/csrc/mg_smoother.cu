// S2: red-black-boundary Gauss-Seidel (gauss_seidel_rbb), NS full sweeps fused into ONE
// pass over memory.  One CTA per tile loads the tile plus a halo of H = 3*NS cells of x, c and the point
// codes into shared memory, then runs red / black / boundary phases entirely on-chip, shrinking the valid
// region by one cell per phase (temporal blocking); halo cells are recomputed redundantly with exactly
// the arithmetic the owning CTA uses, so the result equals NS sequential sweeps bit for bit.
// x is double-buffered (x_in -> x_out): a neighbouring CTA may still be reading the old values.
// HBM traffic per point: x in 8 (0 when x_in is known to be zero) + c 8 + b 8 + lambda 8 + x out 8 + code 2,
// against 64 B per sweep of the three-loop formulation.
#include "mg_device.h"

namespace mgb {

namespace {

constexpr int GT = 512;   // threads per CTA

template <int NS>
struct Geo {
    static constexpr int H = 3 * NS;
    static constexpr int RW = TX + 2 * H;
    static constexpr int RH = TY + 2 * H;
    static constexpr int RN = RW * RH;
};

// global slot of region cell (rx, ry); region origin is (-H, -H) relative to the tile
template <int H>
__device__ __forceinline__ int64_t region_slot(const int* tn, int rx, int ry) {
    const int lx = rx - H, ly = ry - H;
    const int ox = (lx < 0) ? -1 : (lx >= TX ? 1 : 0);
    const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
    return (int64_t)tn[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + (lx - ox * TX);
}

template <int NS>
__global__ void __launch_bounds__(GT) k_gs_fused(LevelDev lv, VecRef xin_r, VecRef xout_r, VecRef b_r, int xin_zero) {
    using G = Geo<NS>;
    constexpr int H = G::H, RW = G::RW, RH = G::RH, RN = G::RN;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sx = reinterpret_cast<double*>(smem_raw);
    double* sc = sx + RN;
    uint16_t* scode = reinterpret_cast<uint16_t*>(sc + RN);
    __shared__ int tn[9];
    const int t = blockIdx.x;
    if (threadIdx.x < 9) tn[threadIdx.x] = lv.tnb[9 * t + threadIdx.x];
    __syncthreads();
    const double* __restrict__ xin = resolve(xin_r);
    double* __restrict__ xout = resolve(xout_r);
    const double* __restrict__ b = resolve(b_r);

    // ---- stage the region
    for (int idx = threadIdx.x; idx < RN; idx += GT) {
        const int ry = idx / RW, rx = idx - ry * RW;
        const int64_t s = region_slot<H>(tn, rx, ry);
        sc[idx] = lv.c[s];
        scode[idx] = lv.code[s];
        sx[idx] = xin_zero ? 0.0 : xin[s];
    }
    __syncthreads();

    const double kappa = lv.kappa;
#pragma unroll 1
    for (int sweep = 0; sweep < NS; sweep++) {
        const int m0 = 3 * sweep;
        // ---- red (colour 0), then black (colour 1): inner points at distance >= m0 + 1 + colour from the edge
#pragma unroll 1
        for (int colour = 0; colour < 2; colour++) {
            const int m = m0 + 1 + colour;
            const int w = RW - 2 * m, hgt = RH - 2 * m;
            const int half = (w + 1) >> 1;
            for (int idx = threadIdx.x; idx < half * hgt; idx += GT) {
                const int row = idx / half, k = idx - row * half;
                const int ry = m + row;
                const int rx = m + 2 * k + ((m + ry + colour) & 1);     // (rx + ry) parity == colour
                if (rx >= RW - m) continue;
                const int p = ry * RW + rx;
                if ((scode[p] & 3) != C_INNER) continue;
                const int64_t s = region_slot<H>(tn, rx, ry);
                const double cl = sc[p];
                const double aW = kappa * (cl + sc[p - 1]), aE = kappa * (cl + sc[p + 1]);
                const double aS = kappa * (cl + sc[p - RW]), aN = kappa * (cl + sc[p + RW]);
                const double all = lv.lam[s] + aW + aE + aS + aN;
                sx[p] = (b[s] + aW * sx[p - 1] + aE * sx[p + 1] + aS * sx[p - RW] + aN * sx[p + RW]) / all;
            }
            __syncthreads();
        }
        // ---- boundary points at distance >= m0 + 3 (Eq. 11, Eq. 16 solved for the point)
        {
            const int m = m0 + 3;
            const int w = RW - 2 * m, hgt = RH - 2 * m;
            for (int idx = threadIdx.x; idx < w * hgt; idx += GT) {
                const int row = idx / w;
                const int ry = m + row, rx = m + (idx - row * w);
                const int p = ry * RW + rx;
                const uint16_t code = scode[p];
                const int kind = code & 3;
                if (kind == C_DIR) {
                    sx[p] = b[region_slot<H>(tn, rx, ry)];
                } else if (kind == C_NEU) {
                    const int tnR = ((code >> 2) & 7) - 2, tnZ = ((code >> 5) & 7) - 2;
                    double sum = 0.0, wself = 0.0, delta;
                    if (code & (1 << 8)) {
                        const int mask = (code >> 9) & 15;
                        if (mask & 1) sum += sx[p - 1];
                        if (mask & 2) sum += sx[p + 1];
                        if (mask & 4) sum += sx[p - RW];
                        if (mask & 8) sum += sx[p + RW];
                        sum = sum / (double)__popc(mask);
                        delta = lv.h;
                    } else {
                        int ox[2], oy[2], nx, ny; double wx, wy;
                        if (tnR & 1) { nx = 2; ox[0] = 0; ox[1] = tnR; wx = 0.5; } else { nx = 1; ox[0] = tnR / 2; ox[1] = 0; wx = 1.0; }
                        if (tnZ & 1) { ny = 2; oy[0] = 0; oy[1] = tnZ; wy = 0.5; } else { ny = 1; oy[0] = tnZ / 2; oy[1] = 0; wy = 1.0; }
                        const double wgt = wx * wy;
                        for (int bb = 0; bb < ny; bb++)
                            for (int aa = 0; aa < nx; aa++) {
                                if (ox[aa] == 0 && oy[bb] == 0) { wself += wgt; continue; }
                                sum += wgt * sx[p + oy[bb] * RW + ox[aa]];
                            }
                        delta = lv.h * sqrt(0.25 * (double)(tnR * tnR + tnZ * tnZ));
                    }
                    sx[p] = (sum - delta * b[region_slot<H>(tn, rx, ry)]) / (1.0 - wself);
                }
            }
            __syncthreads();
        }
    }
    // ---- write the tile back (absent slots carry the zeros they were loaded with)
    for (int idx = threadIdx.x; idx < TS; idx += GT) {
        const int ly = idx / TX, lx = idx - ly * TX;
        xout[(int64_t)t * TS + idx] = sx[(ly + H) * RW + lx + H];
    }
}

__global__ void k_copy(VecRef sr, VecRef dr, int64_t n) {
    const double* __restrict__ s = resolve(sr);
    double* __restrict__ d = resolve(dr);
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) d[k] = s[k];
}

template <int NS>
void launch_ns(const Launch& L, const LevelDev& lv, VecRef xin, VecRef xout, VecRef b, bool zero) {
    constexpr size_t smem = (size_t)Geo<NS>::RN * (2 * sizeof(double) + sizeof(uint16_t));
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_gs_fused<NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = true;
    }
    k_gs_fused<NS><<<lv.ntiles, GT, smem, L.stream>>>(lv, xin, xout, b, zero ? 1 : 0);
}

}  // namespace

void launch_gs_fused(const Launch& L, const LevelDev& lv, VecRef x_in, VecRef x_out, VecRef b, int sweeps, bool x_in_zero) {
    if (sweeps == 2) launch_ns<2>(L, lv, x_in, x_out, b, x_in_zero);
    else launch_ns<1>(L, lv, x_in, x_out, b, x_in_zero);
    if (L.counter) *L.counter += 1;
}

void launch_copy(const Launch& L, VecRef src, VecRef dst, int64_t n) {
    k_copy<<<(int)std::min<int64_t>((n + 255) / 256, 148 * 8), 256, 0, L.stream>>>(src, dst, n);
    if (L.counter) *L.counter += 1;
}

}  // namespace mgb
