// Host-side setup (once per mesh): level point sets, guard classification, Neumann
// stencil codes and the tile tables of the device layout.  Rules M1-M8 and D3 of DESIGN.md section 3.
// Written independently of oracle/: it works on sparse tile bitmaps, not on point lists with
// neighbour indices.
#include "mg_common.h"

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "../../include/mg_b200.h"

namespace mgb {

static inline int64_t tile_key(int64_t TI, int64_t TJ) {
    return ((TJ + (int64_t(1) << 30)) << 31) | (TI + (int64_t(1) << 30));   // |T*| < 2^27: sorts by (TJ, TI)
}

int32_t HostLevel::find_tile(int64_t TI, int64_t TJ) const {
    const int64_t k = tile_key(TI, TJ);
    auto it = std::lower_bound(keys.begin(), keys.end(), k);
    if (it == keys.end() || *it != k) return -1;
    return id_of_key[it - keys.begin()];
}

int64_t HostLevel::slot_of(int64_t I, int64_t J) const {
    const int64_t TI = floordiv(I, TX), TJ = floordiv(J, TY);
    const int32_t t = find_tile(TI, TJ);
    if (t < 0) return -1;
    return (int64_t)t * TS + (J - TJ * TY) * TX + (I - TI * TX);
}

uint16_t HostLevel::get(int64_t I, int64_t J) const {
    const int64_t s = slot_of(I, J);
    return s < 0 ? C_ABSENT : code[s];
}

namespace {

struct Pt { int32_t I, J; uint8_t kind; };
const int DI[4] = {-1, 1, 0, 0}, DJ[4] = {0, 0, -1, 1};   // W, E, S, N

// Creates tiles + codes (kind only) from a point list. Returns false on a duplicate point.
bool fill_level(HostLevel& lv, const std::vector<Pt>& pts, std::vector<int32_t>* slot_out) {
    std::vector<int64_t> k(pts.size());
    for (size_t p = 0; p < pts.size(); p++) k[p] = tile_key(floordiv(pts[p].I, TX), floordiv(pts[p].J, TY));
    lv.keys = k;
    std::sort(lv.keys.begin(), lv.keys.end());
    lv.keys.erase(std::unique(lv.keys.begin(), lv.keys.end()), lv.keys.end());
    lv.ntiles = (int32_t)lv.keys.size();
    lv.tI.resize(lv.ntiles); lv.tJ.resize(lv.ntiles);
    // Tile order = order of the tile ids in memory and in the smoother's work lists.  0: (TJ, TI) row-major (default);
    // 1: Morton (Z-curve) over the tile coordinates; 2: parent-grouped — the 2 x 2 tiles under one coarse tile adjacent,
    // parents row-major.  The paper's ordering study at tile granularity: profiles/r02_layout.md.
    static const int order = getenv("MG_B200_TILE_ORDER") ? atoi(getenv("MG_B200_TILE_ORDER")) : 0;
    std::vector<int32_t> cI(lv.ntiles), cJ(lv.ntiles), pos(lv.ntiles);
    for (int32_t q = 0; q < lv.ntiles; q++) {
        cJ[q] = (int32_t)((lv.keys[q] >> 31) - (int64_t(1) << 30));
        cI[q] = (int32_t)((lv.keys[q] & 0x7fffffffLL) - (int64_t(1) << 30));
    }
    std::iota(pos.begin(), pos.end(), 0);
    if (order != 0 && lv.ntiles > 0) {
        const int32_t i0 = *std::min_element(cI.begin(), cI.end()) & ~1, j0 = *std::min_element(cJ.begin(), cJ.end()) & ~1;
        auto spread = [](uint64_t v) { uint64_t r = 0; for (int b = 0; b < 28; b++) r |= ((v >> b) & 1ull) << (2 * b); return r; };
        std::vector<uint64_t> sk(lv.ntiles);
        for (int32_t q = 0; q < lv.ntiles; q++) {
            const uint64_t a = (uint64_t)(cI[q] - i0), b = (uint64_t)(cJ[q] - j0);
            sk[q] = order == 1 ? (spread(a) | (spread(b) << 1)) : ((((b >> 1) << 28 | (a >> 1)) << 2) | ((b & 1) << 1) | (a & 1));
        }
        std::stable_sort(pos.begin(), pos.end(), [&](int32_t x, int32_t y) { return sk[x] < sk[y]; });
    }
    lv.id_of_key.assign(lv.ntiles, 0);
    for (int32_t id = 0; id < lv.ntiles; id++) { lv.id_of_key[pos[id]] = id; lv.tI[id] = cI[pos[id]]; lv.tJ[id] = cJ[pos[id]]; }
    lv.code.assign((size_t)lv.nslots(), C_ABSENT);
    if (slot_out) slot_out->resize(pts.size());
    lv.n = (int64_t)pts.size(); lv.n_inner = 0;
    for (size_t p = 0; p < pts.size(); p++) {
        const int32_t t = lv.id_of_key[std::lower_bound(lv.keys.begin(), lv.keys.end(), k[p]) - lv.keys.begin()];
        const int64_t s = (int64_t)t * TS + (pts[p].J - (int64_t)lv.tJ[t] * TY) * TX + (pts[p].I - (int64_t)lv.tI[t] * TX);
        if (lv.code[s] != C_ABSENT) return false;
        lv.code[s] = (uint16_t)(pts[p].kind + 1);
        lv.n_inner += (pts[p].kind == 0);
        if (slot_out) (*slot_out)[p] = (int32_t)s;
    }
    return true;
}

inline int psi2(uint16_t c) {                         // Eq. 12 doubled: inner 2, boundary 1, absent 0
    const int k = code_kind(c);
    return k == C_ABSENT ? 0 : (k == C_INNER ? 2 : 1);
}

// Rule D3: encode the discrete normal of every Neumann guard and decide whether
// the bilinear upstream stencil is admissible (all non-self nodes inner) or the fallback is used.
void encode_neumann(HostLevel& lv) {
    for (int32_t t = 0; t < lv.ntiles; t++)
        for (int ly = 0; ly < TY; ly++)
            for (int lx = 0; lx < TX; lx++) {
                const int64_t s = (int64_t)t * TS + ly * TX + lx;
                if (code_kind(lv.code[s]) != C_NEU) continue;
                const int64_t I = (int64_t)lv.tI[t] * TX + lx, J = (int64_t)lv.tJ[t] * TY + ly;
                uint16_t nb[4]; int mask = 0;
                for (int d = 0; d < 4; d++) {
                    nb[d] = lv.get(I + DI[d], J + DJ[d]);
                    if (code_kind(nb[d]) == C_INNER) mask |= 1 << d;
                }
                const int tnR = psi2(nb[1]) - psi2(nb[0]), tnZ = psi2(nb[3]) - psi2(nb[2]);   // Eq. 13 (x2)
                bool fb = (tnR == 0 && tnZ == 0);
                if (!fb) {
                    // per axis: integer n -> offset {n}; half-integer -> offsets {0, 2n} (Eq. 14, 15)
                    int ox[2], oy[2], nx, ny;
                    if (tnR & 1) { nx = 2; ox[0] = 0; ox[1] = tnR; } else { nx = 1; ox[0] = tnR / 2; }
                    if (tnZ & 1) { ny = 2; oy[0] = 0; oy[1] = tnZ; } else { ny = 1; oy[0] = tnZ / 2; }
                    for (int b = 0; b < ny; b++)
                        for (int a = 0; a < nx; a++) {
                            if (ox[a] == 0 && oy[b] == 0) continue;
                            if (code_kind(lv.get(I + ox[a], J + oy[b])) != C_INNER) fb = true;
                        }
                }
                lv.code[s] = (uint16_t)(C_NEU | ((tnR + 2) << 2) | ((tnZ + 2) << 5) | ((fb ? 1 : 0) << 8) | (mask << 9));
            }
}

void build_tile_tables(HostLevel& lv) {
    lv.tnb.assign((size_t)9 * lv.ntiles, lv.ntiles);
    for (int32_t t = 0; t < lv.ntiles; t++)
        for (int dy = -1; dy <= 1; dy++)
            for (int dx = -1; dx <= 1; dx++) {
                const int32_t q = lv.find_tile((int64_t)lv.tI[t] + dx, (int64_t)lv.tJ[t] + dy);
                lv.tnb[(size_t)9 * t + (dy + 1) * 3 + (dx + 1)] = q < 0 ? lv.ntiles : q;
            }
    // interior flags: the smoother's fast path needs every cell within 2 NS (+ 2 with the fused defect
    // restriction) cells of the tile to be an inner point: bits 0, 1, 2 = halo 2, 4, 6 all inner
    lv.tflag.assign((size_t)lv.ntiles + 1, 0);
    for (int32_t t = 0; t < lv.ntiles; t++) {
        int reach = 6;                                       // largest halo (0, 2, 4 or 6) that is all inner
        for (int ly = -6; ly < TY + 6 && reach > 0; ly++)
            for (int lx = -6; lx < TX + 6; lx++) {
                const int dist = std::max(std::max(-lx, lx - (TX - 1)), std::max(-ly, ly - (TY - 1)));   // 0 inside the tile
                if (dist > reach) continue;
                const int ox = lx < 0 ? -1 : (lx >= TX ? 1 : 0), oy = ly < 0 ? -1 : (ly >= TY ? 1 : 0);
                const int32_t q = lv.tnb[(size_t)9 * t + (oy + 1) * 3 + (ox + 1)];
                const uint16_t c = lv.code[(size_t)q * TS + (ly - oy * TY) * TX + (lx - ox * TX)];
                if (code_kind(c) != C_INNER) reach = std::min(reach, dist <= 2 ? 0 : (dist <= 4 ? 2 : 4));
                if (reach == 0) break;
            }
        lv.tflag[t] = (uint8_t)((reach >= 2 ? 1 : 0) | (reach >= 4 ? 2 : 0) | (reach >= 6 ? 4 : 0));
    }
    // tile lists of the register-tiled smoother: interior tiles, general tiles, and tiles with more guards in reach
    // than the smoother's guard list holds
    std::vector<uint8_t> ovf((size_t)lv.ntiles, 0);
    for (int32_t t = 0; t < lv.ntiles; t++) {
        if (lv.tflag[t] & 4) continue;
        int ng = 0;
        for (int ly = -8; ly < TY + 8; ly++)
            for (int lx = -8; lx < TX + 8; lx++) {
                const int ox = lx < 0 ? -1 : (lx >= TX ? 1 : 0), oy = ly < 0 ? -1 : (ly >= TY ? 1 : 0);
                const int32_t q = lv.tnb[(size_t)9 * t + (oy + 1) * 3 + (ox + 1)];
                ng += code_kind(lv.code[(size_t)q * TS + (ly - oy * TY) * TX + (lx - ox * TX)]) >= C_DIR;
            }
        ovf[t] = ng > GUARD_CAP;
    }
    for (int k = 0; k < 2; k++) {
        lv.tlist[k].clear();
        for (int32_t t = 0; t < lv.ntiles; t++) if (lv.tflag[t] & (2 << k)) lv.tlist[k].push_back(t);
        lv.nint[k] = (int32_t)lv.tlist[k].size();
        for (int32_t t = 0; t < lv.ntiles; t++) if (!(lv.tflag[t] & (2 << k)) && !ovf[t]) lv.tlist[k].push_back(t);
        lv.ngen[k] = (int32_t)lv.tlist[k].size() - lv.nint[k];
        for (int32_t t = 0; t < lv.ntiles; t++) if (!(lv.tflag[t] & (2 << k)) && ovf[t]) lv.tlist[k].push_back(t);
    }
    // canonical order: ascending (J, I)
    lv.canon2slot.clear(); lv.canon2slot.reserve((size_t)lv.n);
    int32_t t0 = 0;                                  // positions in `keys` (sorted by (TJ, TI)): one tile row at a time
    while (t0 < lv.ntiles) {
        int32_t t1 = t0;
        while (t1 < lv.ntiles && (lv.keys[t1] >> 31) == (lv.keys[t0] >> 31)) t1++;
        for (int ly = 0; ly < TY; ly++)
            for (int32_t q = t0; q < t1; q++) {
                const int32_t t = lv.id_of_key[q];
                const uint16_t* c = &lv.code[(size_t)t * TS + ly * TX];
                for (int lx = 0; lx < TX; lx++)
                    if (c[lx] != C_ABSENT) lv.canon2slot.push_back((int32_t)((int64_t)t * TS + ly * TX + lx));
            }
        t0 = t1;
    }
}

void build_transfer_tables(HostLevel& f, HostLevel& c) {
    c.ctab.assign((size_t)9 * c.ntiles, f.ntiles);
    for (int32_t t = 0; t < c.ntiles; t++)
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                const int32_t q = f.find_tile(2 * (int64_t)c.tI[t] - 1 + b, 2 * (int64_t)c.tJ[t] - 1 + a);
                c.ctab[(size_t)9 * t + a * 3 + b] = q < 0 ? f.ntiles : q;
            }
    f.ptab.assign((size_t)9 * f.ntiles, c.ntiles);
    for (int32_t t = 0; t < f.ntiles; t++) {
        const int64_t pI = floordiv(f.tI[t], 2), pJ = floordiv(f.tJ[t], 2);   // parent tile
        for (int a = -1; a <= 1; a++)
            for (int b = -1; b <= 1; b++) {
                const int32_t q = c.find_tile(pI + b, pJ + a);
                f.ptab[(size_t)9 * t + (a + 1) * 3 + (b + 1)] = q < 0 ? c.ntiles : q;
            }
    }
}

// Rules M3 (coarse inner = fine inner with even indices), M2 (one guard layer), M4 (type inheritance).
bool coarsen(const HostLevel& f, HostLevel& c) {
    std::vector<Pt> pts;
    for (int32_t t = 0; t < f.ntiles; t++)
        for (int ly = 0; ly < TY; ly += 2)
            for (int lx = 0; lx < TX; lx += 2)      // tile origins are even, so local parity == global parity
                if (code_kind(f.code[(size_t)t * TS + ly * TX + lx]) == C_INNER)
                    pts.push_back({(int32_t)(((int64_t)f.tI[t] * TX + lx) / 2), (int32_t)(((int64_t)f.tJ[t] * TY + ly) / 2), 0});
    if (pts.empty()) return false;
    HostLevel in;                                   // inner-only bitmap for the adjacency tests
    fill_level(in, pts, nullptr);
    const size_t n_in = pts.size();
    std::vector<std::pair<int64_t, int64_t>> cand;  // (J, I) of guard candidates
    for (size_t p = 0; p < n_in; p++)
        for (int d = 0; d < 4; d++) {
            const int64_t gi = (int64_t)pts[p].I + DI[d], gj = (int64_t)pts[p].J + DJ[d];
            if (in.get(gi, gj) == C_ABSENT) cand.push_back({gj, gi});
        }
    std::sort(cand.begin(), cand.end());
    cand.erase(std::unique(cand.begin(), cand.end()), cand.end());
    for (auto& g : cand) {
        const int64_t gj = g.first, gi = g.second;
        bool dirichlet = false;
        for (int e = 0; e < 4; e++) {
            const int64_t qi = gi + DI[e], qj = gj + DJ[e];
            if (in.get(qi, qj) == C_ABSENT) continue;
            const uint16_t mid = f.get(gi + qi, gj + qj);                       // fine midpoint of g and q
            const uint16_t src = (code_kind(mid) == C_INNER) ? f.get(2 * gi, 2 * gj) : mid;
            if (code_kind(src) == C_DIR) dirichlet = true;
        }
        pts.push_back({(int32_t)gi, (int32_t)gj, (uint8_t)(dirichlet ? 1 : 2)});
    }
    c.h = 2.0 * f.h;                                // reading G2 of PAPER.md:151
    fill_level(c, pts, nullptr);
    encode_neumann(c);
    build_tile_tables(c);
    return true;
}

}  // namespace

int build_hierarchy(int64_t n, const int32_t* i, const int32_t* j, const uint8_t* kind, double h, int levels,
                    HostHierarchy& out) {
    out.lev.clear();
    out.lev.reserve(40);
    out.lev.emplace_back();
    HostLevel& l0 = out.lev[0];
    l0.h = h;
    std::vector<Pt> pts((size_t)n);
    for (int64_t p = 0; p < n; p++) {
        if (kind[p] > 2) { out.err = "kind out of range"; return MG_EINVAL; }
        pts[p] = {i[p], j[p], kind[p]};
    }
    if (!fill_level(l0, pts, &out.user2slot)) { out.err = "duplicate (i,j)"; return MG_EMESH; }
    // M2 validation
    for (int64_t p = 0; p < n; p++) {
        bool has_inner = false;
        for (int d = 0; d < 4; d++) {
            const uint16_t c = l0.get((int64_t)i[p] + DI[d], (int64_t)j[p] + DJ[d]);
            if (kind[p] == 0 && c == C_ABSENT) { out.err = "inner point lacks a neighbour"; return MG_EMESH; }
            if (code_kind(c) == C_INNER) has_inner = true;
        }
        if (kind[p] != 0 && !has_inner) { out.err = "guard without inner 4-neighbour"; return MG_EMESH; }
    }
    encode_neumann(l0);
    build_tile_tables(l0);
    const int want = levels > 0 ? levels : 40;
    while ((int)out.lev.size() < want) {
        HostLevel& f = out.lev.back();
        if (levels <= 0) {                          // M8 auto rule
            int64_t imin = INT64_MAX, imax = INT64_MIN, jmin = INT64_MAX, jmax = INT64_MIN;
            for (int32_t t = 0; t < f.ntiles; t++)
                for (int s = 0; s < TS; s++)
                    if (f.code[(size_t)t * TS + s] != C_ABSENT) {
                        const int64_t I = (int64_t)f.tI[t] * TX + s % TX, J = (int64_t)f.tJ[t] * TY + s / TX;
                        imin = std::min(imin, I); imax = std::max(imax, I); jmin = std::min(jmin, J); jmax = std::max(jmax, J);
                    }
            if (std::max(imax - imin + 1, jmax - jmin + 1) <= 9) break;
        }
        HostLevel c;
        if (!coarsen(f, c)) break;
        if (levels <= 0 && c.n_inner < 16) break;
        out.lev.push_back(std::move(c));
        build_transfer_tables(out.lev[out.lev.size() - 2], out.lev.back());
    }
    return MG_OK;
}

}  // namespace mgb
