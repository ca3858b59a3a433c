// Internal definitions shared by the host setup, the kernels and the C-ABI layer of libmg_b200.
// (Nothing here is shared with oracle/.)
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace mgb {

// ---- device tile layout -------------------------------------------------------------------------
// A level's lattice is cut into TX x TY tiles aligned to multiples of (TX, TY) in the level's own
// lattice indices; only tiles holding at least one mesh point are stored ("active tiles"), sorted by
// (TJ, TI).  A vector has (ntiles + 1) * TS slots: slot = tile * TS + ly * TX + lx; the extra tile
// (id = ntiles) is the all-absent "null tile" every missing neighbour points to, so that halo
// addressing needs no branch.  TX and TY are even, hence colour(I + J) == colour(lx + ly) and a
// coarse tile covers exactly 2 x 2 fine tiles.
constexpr int TX = 64;
constexpr int TY = 32;
constexpr int TS = TX * TY;
constexpr int GUARD_CAP = 512;   // capacity of the per-CTA guard list of the smoother kernels

// Per-slot 16-bit code.
//  bits 0-1 : 0 absent, 1 inner, 2 Dirichlet guard, 3 Neumann guard
//  Neumann guards only (rule D3):
//  bits 2-4 : 2 n^R + 2   (0..4)        bits 5-7 : 2 n^Z + 2
//  bit  8   : fallback stencil (mean of inner 4-neighbours, delta = h)
//  bits 9-12: which of W, E, S, N are inner points (used by the fallback)
constexpr uint16_t C_ABSENT = 0, C_INNER = 1, C_DIR = 2, C_NEU = 3;
inline uint16_t code_kind(uint16_t c) { return c & 3; }

inline int64_t floordiv(int64_t a, int64_t b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

struct HostLevel {
    double h = 0;
    int32_t ntiles = 0;
    std::vector<int32_t> tI, tJ;        // tile coordinates per tile id (ids in (TJ, TI) order unless MG_B200_TILE_ORDER says otherwise)
    std::vector<uint16_t> code;         // (ntiles + 1) * TS
    std::vector<int32_t> tnb;           // 9 * ntiles: neighbour tile ids, (dy+1)*3 + (dx+1); missing -> ntiles
    std::vector<int32_t> ctab;          // on a COARSE level: 9 * ntiles ids of the FINE tiles (2TJ-1..2TJ+1) x (2TI-1..2TI+1)
    std::vector<int32_t> ptab;          // on a FINE level: 9 * ntiles ids of the COARSE tiles (pTJ-1..pTJ+1) x (pTI-1..pTI+1), pT = floor(T/2)
    std::vector<uint8_t> tflag;         // per tile: bit 0 / 1 / 2 = all cells within 2 / 4 / 6 cells of the tile are inner points
    // tiles sorted into [interior | general | overflow]: interior by flag bit 1 (k = 0: halo 4) / bit 2 (k = 1: halo 6);
    // overflow = more than GUARD_CAP guard points within 8 cells of the tile (they stay on the shared-memory tile code)
    std::vector<int32_t> tlist[2];
    int32_t nint[2] = {0, 0}, ngen[2] = {0, 0};
    std::vector<int32_t> canon2slot;    // canonical (J, I) order -> slot
    int64_t n = 0, n_inner = 0;
    int64_t nslots() const { return (int64_t)(ntiles + 1) * TS; }
    // lookup
    std::vector<int64_t> keys;          // sorted tile keys for binary search
    std::vector<int32_t> id_of_key;     // position in `keys` -> tile id (the tile ORDER is a layout choice: row-major by default,
                                        // Morton or parent-grouped for the ordering study, MG_B200_TILE_ORDER)
    int32_t find_tile(int64_t TI, int64_t TJ) const;
    uint16_t get(int64_t I, int64_t J) const;     // code at lattice point, 0 if absent
    int64_t slot_of(int64_t I, int64_t J) const;  // -1 if the tile is not active
};

struct HostHierarchy {
    std::vector<HostLevel> lev;
    std::vector<int32_t> user2slot;     // level 0: user point -> slot
    std::string err;
};

// Builds every level from the user's mesh (rules M1-M8, D3 codes, tile tables). Returns 0 or MG_E*.
int build_hierarchy(int64_t n, const int32_t* i, const int32_t* j, const uint8_t* kind, double h, int levels,
                    HostHierarchy& out);

}  // namespace mgb
