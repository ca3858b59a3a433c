// S2 (+S3, S4, S1) on INTERIOR tiles of the large levels, register-tiled: the same two fused red-black Gauss-Seidel
// sweeps (gauss_seidel_rbb; every cell of an interior tile's region is an inner point, so the boundary
// loop is empty), optionally preceded by the coarse-grid correction x <- x - P e_c and followed by the
// restricted defect or by w = A x, as gs_fast of mg_tile_gs.cuh — same arithmetic in the same
// order, so both kernels produce the same bits — but organised around registers instead of shared memory:
//
//   * a thread owns a STRIP: one column pair (2p, 2p+1) x R consecutive rows of the region (tile + halo H).  In every
//     row of a pair exactly one cell is red and one is black, at positions fixed at compile time, so the colour
//     phases are straight-line code over registers: x, b, 1/a_ll and the face sums (c_l + c_nb) of the strip stay in
//     registers for the whole kernel (the face sums are sweep-invariant: computed once), the N/S neighbours and one
//     of the W/E neighbours of every cell are the thread's own registers;
//   * shared memory only carries what crosses a strip boundary: every updated value is also published to a
//     colour-split mirror of x (the layout of mg_tile_gs.cuh), from which a thread reads the ONE cross-lane W/E
//     neighbour of each cell and the rows just above / below its strip.  Per cell update: 1 LDS.64 + 1 STS.64 (+ 2 LDS
//     per strip and phase) against 9 LDS.64 + 1 STS.64 in gs_fast;
//   * a warp of "main" strips covers exactly the 32 column pairs of the tile, one warp per block of R rows, so its
//     global loads and stores are whole 512-byte tile rows (LDG.128 / STG.128).  The H halo column pairs of the row
//     blocks are packed into a few extra warps (32 / H row blocks per warp);
//   * no predication: every strip runs every phase; values within p cells of the region edge are wrong after phase p
//     and never reach the tile (halo H >= 2 NS), as in any temporally blocked sweep;
//   * the CTA is persistent (one per SM: the register file holds one region) and walks a list of interior tiles.
//     Loads are decoupled from the arithmetic by asynchronous copies (cp.async, SASS LDGSTS): while tile i is swept in
//     registers, every thread's strip of tile i + 1 (x, c, b, 1/a_ll, lambda, coarse parents) streams from HBM into
//     that thread's PRIVATE staging slots in shared memory — private, so no barrier guards the staging buffer and one
//     buffer suffices: a thread refills its slots right after it has moved them into registers.  The per-tile tables
//     (neighbour tiles, parent tiles) come from a packed per-list array two tiles ahead.
//
// GEN = true is the same kernel for tiles whose region contains guard or absent cells (gs_general of mg_tile_gs.cuh):
// the halo grows by one cell per sweep for the boundary loop of gauss_seidel_rbb, every strip carries a
// mask of its inner cells (the others keep their value in the colour phases), the guard cells of the region are
// collected once into a list and updated from the mirror after each black phase (Eq. 11 / Eq. 16 solved for the
// point), and their owners reload them.  Tiles with more guards in reach than the list holds stay on k_gs.
#pragma once
#include "mg_tile_gs.cuh"

namespace mgb {
namespace {

template <int H>
struct SGeo {
    static_assert(H % 2 == 0 && 32 % 1 == 0, "halo must be even: column pairs may not straddle tiles");
    static constexpr int R = 4;                          // rows per strip
    static constexpr int RW = TX + 2 * H, RH = TY + 2 * H, RWC = RW / 2;
    static_assert(RH % R == 0, "region height must be a multiple of the strip height");
    static constexpr int NRB = RH / R;                   // row blocks = main warps
    static constexpr int RBL = 32 / H;                   // row blocks of halo pairs per extra warp
    static constexpr int NLW = (NRB + RBL - 1) / RBL;    // extra warps
    static constexpr int NW = NRB + NLW, NT = 32 * NW;
    static constexpr int NCP = (RH + 2) * RWC;           // cells per colour, one padding row below and above the region
    static constexpr size_t MIRROR = (size_t)4 * NCP * sizeof(double);   // mirrors of x and c (c: later d / w scratch)
    // + staging: NA arrays x R rows x NT threads of 16-byte pairs, (PC) 6 coarse values per thread, 3 tile-table buffers
    static constexpr int NA = 2;
    // geometry handed to neumann_smem / cidx of mg_tile_gs.cuh (mirror pointer advanced by the padding row)
    static constexpr int NC = NCP;
    static constexpr size_t smem(bool pc, bool gen) {
        return MIRROR + (size_t)NA * R * NT * 16 + (pc ? (size_t)6 * NT * 8 : 0) + 3 * 24 * 4 +
               (gen ? (size_t)R * NT * 4 + (size_t)GCAP * 12 : 0);
    }
};
constexpr int SMETA = 24;   // ints per list entry of LevelDev::smeta: tn[9], pt[9], odd[2], tile id, padding

__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async8(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void prefetch_l2_bulk(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// x_out = S^NS (x_in - [PC] P e_c), NS = 1 or 2 sweeps, on the nlist tiles described by smeta; EPI as in k_gs (1: d_c = R (A x_out - b), 2: w = A x_out).
// CTA `cta` of `ncta` walks the list entries cta, cta + ncta, ...; barriers count the NT threads of this geometry only
// (the launch may carry more: the two geometries of k_gs_strip share one grid).
template <int NTHREADS>
__device__ __forceinline__ void bar_sync() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }

// XI: the three-field form (Eq. 3): the smoother works on the row divided by xi — it holds b / xi, and 1/a_ll is
// xi / a_ll (k_diag) — and the epilogues scale kappa by xi of the row's point, exactly as mg_tile_gs.cuh does.
template <int NS, int H, bool PC, int EPI, bool GEN, bool MP, bool XI>
__device__ __forceinline__ void strip_body(const LevelDev& lv, const int* __restrict__ smeta, int nlist, int planes, const VecRef& xin_r,
                                           const VecRef& xout_r, const VecRef& b_r, const double* __restrict__ ec0, int xin_zero,
                                           const uint16_t* __restrict__ ccode, double* __restrict__ dc0, const int* __restrict__ stop, int cta,
                                           int ncta, unsigned char* smem_raw) {
    using G = SGeo<H>;
    constexpr int R = G::R, RWC = G::RWC, NCP = G::NCP, NRB = G::NRB, RBL = G::RBL, NT = G::NT;
    constexpr bool DR = EPI == 1, AP = EPI == 2;
    constexpr int NA = SGeo<H>::NA;                         // staged arrays: c, x (b, 1/a_ll, lambda: loaded directly, after an L2 prefetch)
    // the valid region shrinks by one cell per phase: two per sweep on interior tiles, three (red, black, boundary) on general ones
    static_assert(H >= (GEN ? 3 * NS + (PC ? 1 : 0) : 2 * NS) + (DR ? 2 : (AP ? 1 : 0)), "halo too small for NS sweeps and the epilogue");
    if ((int)threadIdx.x >= NT) return;
    double* sx = reinterpret_cast<double*>(smem_raw);       // [2][RH + 2][RWC] colour-split mirror of x
    double* sc = sx + 2 * NCP;                              // same for c; dead after the face sums: scratch of the epilogues
    double2* stg = reinterpret_cast<double2*>(sc + 2 * NCP);   // [NA][R][NT] private staging slots
    double* se = reinterpret_cast<double*>(stg + NA * R * NT); // (PC) [6][NT] coarse parents
    int* M = reinterpret_cast<int*>(se + (PC ? 6 * NT : 0));   // [3][SMETA] tile tables of tiles i, i + 1, i + 2
    uint32_t* cstg = reinterpret_cast<uint32_t*>(M + 3 * SMETA);                 // (GEN) [R][NT] staged point codes of the pairs
    double* gb = reinterpret_cast<double*>(cstg + (GEN ? R * NT : 0));           // (GEN) guard list: right-hand side,
    uint16_t* gcell = reinterpret_cast<uint16_t*>(gb + (GEN ? GCAP : 0));        //       cell ry * RW + rx,
    uint16_t* gcode = gcell + (GEN ? GCAP : 0);                                  //       point code
    __shared__ int gcount;
    double* sxp = sx + RWC;                                 // mirror as neumann_smem / cidx<G> address it (region row 0 = padded row 1)
    // work items: (plane, list entry) pairs, plane-major; the vectors of plane pl (one solve per plane, same mesh)
    struct PP { const double *c, *rd, *lam, *xi, *b, *xin, *ec; double *xout, *dc; };
    auto plane_ptrs = [&](int pl) {
        const int64_t po = (int64_t)pl * lv.nslots, pco = (int64_t)pl * (lv.ntiles_coarse + 1) * TS;
        PP q;
        q.c = lv.c + po; q.rd = lv.rd + po; q.lam = lv.lam + po; q.xi = XI ? lv.xi + po : nullptr;
        q.b = resolve(b_r, pl); q.xin = resolve(xin_r, pl); q.xout = resolve(xout_r, pl);
        q.ec = PC ? ec0 + pco : nullptr;
        q.dc = DR ? dc0 + pco : (AP ? dc0 + po : nullptr);
        return q;
    };
    const int nitems = MP ? nlist * planes : nlist;       // MP: several planes in the launch (pointers per work item)
    const PP one = plane_ptrs(0);
    if (cta >= nitems) return;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // ---- the strip of this thread: pair column p, rows ry0 .. ry0 + R - 1 of the region
    int p, rb;
    const bool main_w = warp < NRB;
    bool spare = false;
    if (main_w) { p = H / 2 + lane; rb = warp; }
    else {
        int g = lane / H, k = lane - g * H;
        rb = (warp - NRB) * RBL + g;
        if (g >= RBL || rb >= NRB) { g = 0; k = 0; rb = (warp - NRB) * RBL; spare = true; }   // spare lanes duplicate the warp's first strip
        p = (k < H / 2) ? k : 32 + k;
    }
    const int ry0 = rb * R;
    const int lx0 = 2 * p - H;                              // tile-relative column of the pair's first cell (even)
    const int ox = (lx0 < 0) ? -1 : (lx0 >= TX ? 1 : 0);
    const int lxm = lx0 - ox * TX;
    // colour-split index of cell (pos, row r) of the strip: colour (r + pos) & 1 (ry0, 2p even), row ry0 + r + 1 (padding), column p
    const int sbase = (ry0 + 1) * RWC + p;
#define SIDX(pos, r) ((((r) + (pos)) & 1) * NCP + sbase + (r) * RWC)
    const double kappa = lv.kappa;
    const int G0 = ncta;

    // asynchronous copies of this thread's strip of the tile described by m[] into its staging slots
    auto prefetch = [&](const int* m) {
        if (MP && m[22]) { cp_async_commit(); return; }      // the plane of that item has ended its cycle: nothing to do
        const PP q = MP ? plane_ptrs(m[21]) : one;
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int ly = ry0 + r - H;
            const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
            const int64_t gs = (int64_t)m[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + lxm;
            cp_async16(&stg[(0 * R + r) * NT + tid], q.c + gs);
            if (!xin_zero) cp_async16(&stg[(1 * R + r) * NT + tid], q.xin + gs);
            if (GEN) cp_async4(&cstg[r * NT + tid], lv.code + gs);
        }
        if (tid < 4) {                                       // b, 1/a_ll, lambda, xi of that tile: into L2 now, into registers when its turn comes
            const int64_t o = (int64_t)m[20] * TS;
            const double* src = tid == 0 ? q.b + o : (tid == 1 ? q.rd + o : (tid == 2 ? (EPI ? q.lam + o : nullptr) : (XI ? q.xi + o : nullptr)));
            if (src != nullptr) prefetch_l2_bulk(src, TS * sizeof(double));
        }
        if (PC) {
            // coarse parents of the strip (bilinear prolongation): columns cx, cx + 1, rows cy0 .. cy0 + 2
            const int cx = m[18] * (TX / 2) + (lx0 >> 1), cy0 = m[19] * (TY / 2) + ((ry0 - H) >> 1);
#pragma unroll
            for (int k = 0; k < 3; k++) {
                cp_async8(&se[(2 * k) * NT + tid], q.ec + parent_slot9(m + 9, cx, cy0 + k));
                cp_async8(&se[(2 * k + 1) * NT + tid], q.ec + parent_slot9(m + 9, cx + 1, cy0 + k));
            }
        }
        cp_async_commit();
    };

    // right-hand sides of the collected guards (the list is complete: call after a barrier), read by the boundary phases
    auto fill_gb = [&](const int* m, const double* __restrict__ b) {
        const int ng = min(gcount, GCAP);
        for (int g = tid; g < ng; g += NT) {
            const int cell = gcell[g], ry = cell / G::RW, rx = cell - ry * G::RW;
            gb[g] = __ldg(b + region_slot<H>(m, rx, ry));
        }
    };
    // table entry `tid` of work item `item`: the list entry's tables, [21] its plane, [22] whether that plane has stopped
    auto meta_of = [&](int item) {
        const int pl = MP ? item / nlist : 0, e = item - pl * nlist;
        if (tid == 21) return pl;
        if (tid == 22) return (MP && stopped(stop, pl)) ? 1 : 0;
        return __ldg(smeta + (int64_t)e * SMETA + tid);
    };

    if (tid == 0) gcount = 0;
    if (tid < SMETA) {
        M[tid] = meta_of(cta);
        if (cta + G0 < nitems) M[SMETA + tid] = meta_of(cta + G0);
    }
    bar_sync<NT>();
    prefetch(M);
    int ib = 0;                                             // buffer of the current tile's tables
    for (int it = cta; it < nitems; it += G0) {
        const int* m = M + ib * SMETA;
        const int* pt = m + 9;
        const int* odd = m + 18;
        const int t = m[20];
        const bool more2 = it + 2 * G0 < nitems;
        int mnext = 0;
        if (tid < SMETA && more2) mnext = meta_of(it + 2 * G0);    // tables two tiles ahead
        // ---- the strip: staging slots -> registers (pairs)
        cp_async_wait_all();
        if (MP && m[22]) {                                    // this plane's cycle has ended: keep the pipeline moving, skip the tile
            if (it + G0 < nitems) prefetch(M + (ib == 2 ? 0 : ib + 1) * SMETA);
            if (tid < SMETA && more2) M[(ib == 0 ? 2 : ib - 1) * SMETA + tid] = mnext;
            ib = ib == 2 ? 0 : ib + 1;
            bar_sync<NT>();
            continue;
        }
        const PP cur = MP ? plane_ptrs(m[21]) : one;
        const double* __restrict__ b = cur.b;
        double* __restrict__ xout = cur.xout;
        double* __restrict__ dc = cur.dc;
        double x[R][2], c[R][2], br[R][2], rd[R][2], lam[R][2];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const double2 cv = stg[(0 * R + r) * NT + tid];
            c[r][0] = cv.x; c[r][1] = cv.y;
            if (xin_zero) { x[r][0] = 0.0; x[r][1] = 0.0; }
            else { const double2 xv = stg[(1 * R + r) * NT + tid]; x[r][0] = xv.x; x[r][1] = xv.y; }
        }
        unsigned cinner = 3u;                                 // (DR) bit r / 2: the coarse point under cell 0 of row r is an inner point
        if (DR && GEN && main_w && pt[4] != lv.ntiles_coarse) {
            cinner = 0u;
#pragma unroll
            for (int r = 0; r < R; r += 2) {
                const int ly = ry0 + r - H;
                if (ly >= 0 && ly < TY)
                    cinner |= ((__ldg(ccode + (int64_t)pt[4] * TS + (odd[1] * (TY / 2) + (ly >> 1)) * TX + odd[0] * (TX / 2) + lane) & 3) == C_INNER ? 1u : 0u) << (r >> 1);
            }
        }
        unsigned imask = 0xffu, gmask = 0u;                   // bit 2 r + pos: the cell is an inner point / a guard
        uint32_t cpair[R];
        if (GEN) {
            imask = 0u;
#pragma unroll
            for (int r = 0; r < R; r++) {
                cpair[r] = cstg[r * NT + tid];
#pragma unroll
                for (int q = 0; q < 2; q++) {
                    const unsigned kind = (cpair[r] >> (16 * q)) & 3u;
                    imask |= (kind == C_INNER ? 1u : 0u) << (2 * r + q);
                    gmask |= (kind >= C_DIR ? 1u : 0u) << (2 * r + q);
                }
            }
        }
#pragma unroll
        for (int r = 0; r < R; r++) {                         // first used after the face sums / in the epilogue
            const int ly = ry0 + r - H;
            const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
            const int64_t gs = (int64_t)m[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + lxm;
            const double2 bv = ldg2(b + gs), dv = ldg2(cur.rd + gs);
            br[r][0] = bv.x; br[r][1] = bv.y; rd[r][0] = dv.x; rd[r][1] = dv.y;
            if (XI) {                                         // inner rows are divided by xi; guards keep their b
                const double2 xv2 = ldg2(cur.xi + gs);
                if (!GEN || ((imask >> (2 * r)) & 1u)) br[r][0] = __ddiv_rn(br[r][0], xv2.x);
                if (!GEN || ((imask >> (2 * r + 1)) & 1u)) br[r][1] = __ddiv_rn(br[r][1], xv2.y);
            }
            if (EPI && !GEN) { const double2 lv2 = ldg2(cur.lam + gs); lam[r][0] = lv2.x; lam[r][1] = lv2.y; }
        }
        double e[3][2];
        if (PC) {
#pragma unroll
            for (int q = 0; q < 3; q++) { e[q][0] = se[(2 * q) * NT + tid]; e[q][1] = se[(2 * q + 1) * NT + tid]; }
        }
        // the slots are consumed: refill them with the next tile of this CTA while this one is computed
        if (it + G0 < nitems) prefetch(M + (ib == 2 ? 0 : ib + 1) * SMETA);
        if (GEN && gmask != 0u && !spare) {
            // guards of the region, collected once: Eq. 11 / Eq. 16 need their right-hand side and their point code
#pragma unroll
            for (int r = 0; r < R; r++)
#pragma unroll
                for (int q = 0; q < 2; q++)
                    if ((gmask >> (2 * r + q)) & 1u) {
                        const int pos = atomicAdd(&gcount, 1);
                        if (pos < GCAP) { gcell[pos] = (uint16_t)((ry0 + r) * G::RW + 2 * p + q); gcode[pos] = (uint16_t)(cpair[r] >> (16 * q)); }
                    }
        }
        if (PC) {
            // x <- x - P e_c (bilinear): weights 1 / (1/2, 1/2) / (1/4 x 4) over the parents
            // (cx, cy), (cx+1, cy), (cx, cy+1), (cx+1, cy+1); rows r = 0..3 of the strip use coarse rows cy0 .. cy0 + 2
            double ee[R][2];
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int q = r >> 1;
                if ((r & 1) == 0) {
                    ee[r][0] = e[q][0];
                    ee[r][1] = 0.5 * e[q][0] + 0.5 * e[q][1];
                } else {
                    ee[r][0] = 0.5 * e[q][0] + 0.5 * e[q + 1][0];
                    ee[r][1] = 0.25 * e[q][0] + 0.25 * e[q][1] + 0.25 * e[q + 1][0] + 0.25 * e[q + 1][1];
                }
            }
            if (GEN) {
                // set_bnds_hom: e = 0 on Dirichlet guards, the homogeneous Eq. 16 on Neumann guards, from
                // the inner values of e in the mirror; absent cells carry 0
#pragma unroll
                for (int r = 0; r < R; r++)
#pragma unroll
                    for (int q = 0; q < 2; q++) {
                        if (!((imask >> (2 * r + q)) & 1u)) ee[r][q] = 0.0;
                        sx[SIDX(q, r)] = ee[r][q];
                    }
                bar_sync<NT>();
                fill_gb(m, b);
                const int ng = min(gcount, GCAP);
                for (int g = tid; g < ng; g += NT) {
                    const uint16_t code = gcode[g];
                    if ((code & 3) != C_NEU) continue;
                    const int cell = gcell[g], ry = cell / G::RW, rx = cell - ry * G::RW;
                    if (rx >= 1 && rx < G::RW - 1 && ry >= 1 && ry < G::RH - 1) {
                        double sum, wself, delta;
                        neumann_smem<G>(code, rx, ry, sxp, lv.h, sum, wself, delta);
                        sxp[cidx<G>(rx, ry)] = sum / (1.0 - wself);
                    }
                }
                bar_sync<NT>();
                if (gmask != 0u) {
#pragma unroll
                    for (int r = 0; r < R; r++)
#pragma unroll
                        for (int q = 0; q < 2; q++)
                            if ((gmask >> (2 * r + q)) & 1u) ee[r][q] = sx[SIDX(q, r)];
                }
                bar_sync<NT>();                                // the mirror is about to receive x
            }
#pragma unroll
            for (int r = 0; r < R; r++) { x[r][0] -= ee[r][0]; x[r][1] -= ee[r][1]; }
        }
#pragma unroll
        for (int r = 0; r < R; r++) {
            sx[SIDX(0, r)] = x[r][0]; sx[SIDX(1, r)] = x[r][1];
            sc[SIDX(0, r)] = c[r][0]; sc[SIDX(1, r)] = c[r][1];
        }
        bar_sync<NT>();
        if (GEN && !PC) fill_gb(m, b);
        // ---- face sums c_l + c_nb (sweep-invariant): hW | cell 0 | hM | cell 1 | hE per row, v[r] below row r per column
        double hW[R], hM[R], hE[R], v[R + 1][2];
#pragma unroll
        for (int r = 0; r < R; r++) {
            hW[r] = c[r][0] + sc[SIDX(1, r) - 1];            // W of cell 0: cell 1 of pair p - 1 (other colour, same row)
            hM[r] = c[r][0] + c[r][1];
            hE[r] = c[r][1] + sc[SIDX(0, r) + 1];            // E of cell 1: cell 0 of pair p + 1
        }
#pragma unroll
        for (int q = 0; q < 2; q++) {
            v[0][q] = c[0][q] + sc[SIDX(q, -1)];
#pragma unroll
            for (int r = 1; r < R; r++) v[r][q] = c[r][q] + c[r - 1][q];
            v[R][q] = c[R - 1][q] + sc[SIDX(q, R)];
        }
        // ---- two sweeps: red (colour 0), black (colour 1); the cell of colour col in row r is at position (r + col) & 1
#pragma unroll
        for (int ph = 0; ph < 2 * NS; ph++) {
            const int col = ph & 1;
            const double xs = sx[SIDX(col, -1)];             // S neighbour of the updated cell of row 0 (position col)
            const double xn = sx[SIDX(1 - col, R)];          // N neighbour of the updated cell of row R - 1 (R even: position 1 - col)
            double xc[R];                                    // the cross-lane W / E neighbours
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int pos = (r + col) & 1;
                xc[r] = pos == 0 ? sx[SIDX(1, r) - 1] : sx[SIDX(0, r) + 1];
            }
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int pos = (r + col) & 1;
                const double xW = pos == 0 ? xc[r] : x[r][0], xE = pos == 0 ? x[r][1] : xc[r];
                const double aW = pos == 0 ? hW[r] : hM[r], aE = pos == 0 ? hM[r] : hE[r];
                const double xS = r == 0 ? xs : x[r - 1][pos], xN = r == R - 1 ? xn : x[r + 1][pos];
                double acc = aW * xW;
                acc = fma(aE, xE, acc);
                acc = fma(v[r][pos], xS, acc);
                acc = fma(v[r + 1][pos], xN, acc);
                const double xnew = fma(kappa, acc, br[r][pos]) * rd[r][pos];
                x[r][pos] = (!GEN || ((imask >> (2 * r + pos)) & 1u)) ? xnew : x[r][pos];
            }
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int pos = (r + col) & 1;
                sx[SIDX(pos, r)] = x[r][pos];
            }
            bar_sync<NT>();
            if (GEN && col == 1) {
                // ---- boundary points (third loop of gauss_seidel_rbb): Eq. 11, Eq. 16 solved for the point
                const int ng = min(gcount, GCAP);
                for (int g = tid; g < ng; g += NT) {
                    const uint16_t code = gcode[g];
                    const int cell = gcell[g], ry = cell / G::RW, rx = cell - ry * G::RW;
                    if ((code & 3) == C_DIR) sxp[cidx<G>(rx, ry)] = gb[g];
                    else {
                        double sum, wself, delta;
                        neumann_smem<G>(code, rx, ry, sxp, lv.h, sum, wself, delta);
                        sxp[cidx<G>(rx, ry)] = neumann_point(sum, delta, gb[g], wself);
                    }
                }
                bar_sync<NT>();
                if (gmask != 0u) {
#pragma unroll
                    for (int r = 0; r < R; r++)
#pragma unroll
                        for (int q = 0; q < 2; q++)
                            if ((gmask >> (2 * r + q)) & 1u) x[r][q] = sx[SIDX(q, r)];
                }
            }
        }
        if (EPI && GEN) {                                     // (registers are scarce on this path: lambda only now; it sits in L2)
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int ly = ry0 + r - H;
                const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
                const double2 lv2 = ldg2(cur.lam + (int64_t)m[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + lxm);
                lam[r][0] = lv2.x; lam[r][1] = lv2.y;
            }
        }
        double xi2[R][2];
        if (XI && EPI) {                                      // xi of the strip again for the epilogue (in L2; no register held it through the sweeps)
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int ly = ry0 + r - H;
                const int oy = (ly < 0) ? -1 : (ly >= TY ? 1 : 0);
                const double2 xv2 = ldg2(cur.xi + (int64_t)m[(oy + 1) * 3 + ox + 1] * TS + (ly - oy * TY) * TX + lxm);
                xi2[r][0] = xv2.x; xi2[r][1] = xv2.y;
            }
        }
        // ---- write the tile rows of the main strips
        if (main_w) {
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int ly = ry0 + r - H;
                if (ly >= 0 && ly < TY)
                    *reinterpret_cast<double2*>(xout + (int64_t)t * TS + ly * TX + 2 * lane) = make_double2(x[r][0], x[r][1]);
            }
        }
        if (DR) {
            // d = A x - b (difference form of rule D1) on the RED cells of the tile and of the one-cell ring around it: the
            // black cells were updated last from the current red values, their defect is zero up to rounding
            // (GEN: next to guards the black defects do not vanish: both colours, inner cells only, rule T2)
            const double xsd[2] = {sx[SIDX(0, -1)], sx[SIDX(1, -1)]}, xnd[2] = {sx[SIDX(0, R)], sx[SIDX(1, R)]};
#pragma unroll
            for (int r = 0; r < R; r++)
#pragma unroll
                for (int qq = 0; qq < (GEN ? 2 : 1); qq++) {
                    const int pos = (r + qq) & 1, ry = ry0 + r, rx = 2 * p + pos;
                    double d = 0.0;
                    if ((!GEN || ((imask >> (2 * r + pos)) & 1u)) && min(min(rx, G::RW - 1 - rx), min(ry, G::RH - 1 - ry)) >= H - 1) {
                        const double xl = x[r][pos];
                        const double xW = pos == 0 ? sx[SIDX(1, r) - 1] : x[r][0], xE = pos == 0 ? x[r][1] : sx[SIDX(0, r) + 1];
                        const double xS = r == 0 ? xsd[pos] : x[r - 1][pos], xN = r == R - 1 ? xnd[pos] : x[r + 1][pos];
                        // __dmul_rn: never contracted, so that this kernel and mg_tile_gs.cuh round identically
                        const double kap = XI ? __dmul_rn(kappa, xi2[r][pos]) : kappa, bl = XI ? __dmul_rn(br[r][pos], xi2[r][pos]) : br[r][pos];
                        const double aW = kap * (pos == 0 ? hW[r] : hM[r]), aE = kap * (pos == 0 ? hM[r] : hE[r]);
                        const double aS = kap * v[r][pos], aN = kap * v[r + 1][pos];
                        d = __dsub_rn(row_d1(lam[r][pos], xl, aW, xW, aE, xE, aS, xS, aN, xN), bl);
                    }
                    sc[SIDX(pos, r)] = d;
                }
            bar_sync<NT>();
            // the 32 x 16 coarse points under the tile gather their full-weighting stencils (rule T2; only the red
            // entries are non-zero): coarse point under fine cell 0 of pair p in an even row
            const int ptile = pt[4];
            if (main_w && ptile != lv.ntiles_coarse) {
#pragma unroll
                for (int r = 0; r < R; r += 2) {
                    const int ly = ry0 + r - H;
                    if (ly >= 0 && ly < TY) {
                        const int i0 = SIDX(0, r);               // red cell (2p, ry); diagonal reds: cells 1 of pairs p - 1, p in rows ry -+ 1
                        const int j0 = SIDX(1, r);               // same position in the black array: cell (2p + 1, ry)
                        const int64_t cs = (int64_t)ptile * TS + (odd[1] * (TY / 2) + (ly >> 1)) * TX + odd[0] * (TX / 2) + lane;
                        double acc = 0.0;
                        if (!GEN) {
                            acc += 0.0625 * sc[i0 - RWC - 1];
                            acc += 0.0625 * sc[i0 - RWC];
                            acc += 0.25 * sc[i0];
                            acc += 0.0625 * sc[i0 + RWC - 1];
                            acc += 0.0625 * sc[i0 + RWC];
                        } else if ((cinner >> (r >> 1)) & 1u) {                // coarse guard rows: 0
                            acc += 0.0625 * sc[i0 - RWC - 1];                // (2p - 1, ry - 1)
                            acc += 0.125 * sc[j0 - RWC];                     // (2p,     ry - 1): black array, row ry - 1, column p
                            acc += 0.0625 * sc[i0 - RWC];                    // (2p + 1, ry - 1)
                            acc += 0.125 * sc[j0 - 1];                       // (2p - 1, ry)
                            acc += 0.25 * sc[i0];
                            acc += 0.125 * sc[j0];                           // (2p + 1, ry)
                            acc += 0.0625 * sc[i0 + RWC - 1];
                            acc += 0.125 * sc[j0 + RWC];
                            acc += 0.0625 * sc[i0 + RWC];
                        }
                        dc[cs] = acc;
                    }
                }
            }
        }
        if (AP) {
            // w = A x_out on the tile (rule D1, difference form), both colours
            if (main_w) {
                const double xs0 = sx[SIDX(0, -1)], xs1 = sx[SIDX(1, -1)], xn0 = sx[SIDX(0, R)], xn1 = sx[SIDX(1, R)];
#pragma unroll
                for (int r = 0; r < R; r++) {
                    const int ly = ry0 + r - H;
                    if (ly >= 0 && ly < TY) {
                        const double x0 = x[r][0], x1 = x[r][1];
                        const double xW = sx[SIDX(1, r) - 1], xE = sx[SIDX(0, r) + 1];
                        const double s0 = r == 0 ? xs0 : x[r - 1][0], n0 = r == R - 1 ? xn0 : x[r + 1][0];
                        const double s1 = r == 0 ? xs1 : x[r - 1][1], n1 = r == R - 1 ? xn1 : x[r + 1][1];
                        const double k0 = XI ? __dmul_rn(kappa, xi2[r][0]) : kappa, k1 = XI ? __dmul_rn(kappa, xi2[r][1]) : kappa;
                        const double w0 = row_d1(lam[r][0], x0, k0 * hW[r], xW, k0 * hM[r], x1, k0 * v[r][0], s0, k0 * v[r + 1][0], n0);
                        const double w1 = row_d1(lam[r][1], x1, k1 * hM[r], x0, k1 * hE[r], xE, k1 * v[r][1], s1, k1 * v[r + 1][1], n1);
                        *reinterpret_cast<double2*>(dc + (int64_t)t * TS + ly * TX + 2 * lane) =
                            make_double2((!GEN || ((imask >> (2 * r)) & 1u)) ? w0 : 0.0, (!GEN || ((imask >> (2 * r + 1)) & 1u)) ? w1 : 0.0);
                    }
                }
            }
            if (GEN) {
                // guard rows of the tile (Eq. 11: x; Eq. 16: (phi^N - x) / delta), after the strips' pair stores
                bar_sync<NT>();
                const int ng = min(gcount, GCAP);
                for (int g = tid; g < ng; g += NT) {
                    const uint16_t code = gcode[g];
                    const int cell = gcell[g], ry = cell / G::RW, rx = cell - ry * G::RW;
                    const int lx = rx - H, ly = ry - H;
                    if (lx < 0 || lx >= TX || ly < 0 || ly >= TY) continue;
                    const double xl = sxp[cidx<G>(rx, ry)];
                    double val = xl;
                    if ((code & 3) == C_NEU) {
                        double sum, wself, delta;
                        neumann_smem<G>(code, rx, ry, sxp, lv.h, sum, wself, delta);
                        val = (sum + wself * xl - xl) / delta;
                    }
                    dc[(int64_t)t * TS + ly * TX + lx] = val;
                }
            }
        }
        if (tid < SMETA && more2) M[(ib == 0 ? 2 : ib - 1) * SMETA + tid] = mnext;   // buffer of tile i - 1 = buffer of tile i + 2
        if (GEN) { bar_sync<NT>(); if (tid == 0) gcount = 0; }                        // every reader of the guard list is done
        ib = ib == 2 ? 0 : ib + 1;
        bar_sync<NT>();                                    // the mirrors are free, the tables of tile i + 2 are visible
    }
#undef SIDX
}

// One launch, two geometries: CTAs [0, ggen) run the general tiles (list smeta_g), the others the interior tiles
// (list smeta_i); both persistent, both with their own thread count (the block carries the larger one).
template <int NS, int HI, int HG, bool PC, int EPI, bool MP, bool XI>
__global__ void __launch_bounds__((SGeo<HI>::NT > SGeo<HG>::NT ? SGeo<HI>::NT : SGeo<HG>::NT), 1)
    k_gs_strip(LevelDev lv, const int* __restrict__ smeta_i, int nint, const int* __restrict__ smeta_g, int ngen, int ggen, int planes, VecRef xin_r,
               VecRef xout_r, VecRef b_r, const double* __restrict__ ec, int xin_zero, const uint16_t* __restrict__ ccode,
               double* __restrict__ dc, const int* __restrict__ stop) {
    extern __shared__ __align__(16) unsigned char strip_smem[];
    if (!MP && stopped(stop, 0)) return;
    if ((int)blockIdx.x < ggen) strip_body<NS, HG, PC, EPI, true, MP, XI>(lv, smeta_g, ngen, planes, xin_r, xout_r, b_r, ec, xin_zero, ccode, dc, stop, blockIdx.x, ggen, strip_smem);
    else strip_body<NS, HI, PC, EPI, false, MP, XI>(lv, smeta_i, nint, planes, xin_r, xout_r, b_r, ec, xin_zero, ccode, dc, stop, blockIdx.x - ggen, gridDim.x - ggen, strip_smem);
}

}  // namespace
}  // namespace mgb
