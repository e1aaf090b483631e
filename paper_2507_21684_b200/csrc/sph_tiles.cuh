// sph_tiles.cuh -- the cell-block ("tile") decomposition shared by the neighbour search and the pair kernels.
//
// A tile is an aligned block of B^d cells (B = 1, 2 or 4).  Because the particles are sorted by the Morton key
// of their cell, the rows of a tile are ONE contiguous range of the sorted arrays.  Every neighbour of a row
// of the tile lives in the (B+2)^d halo cells around it; each halo cell is a contiguous run of the sorted arrays.
// The halo cells are numbered in (z,y,x) slot order and their particles concatenated in that order: the
// "halo-linear" index q of a particle.  The 3 cells of a row's neighbour cells that are adjacent along x are
// therefore ONE run of consecutive q, and a row's candidate sequence is 3^(d-1) such runs.
//
// Tile-local lists (PAPER.md:163 pair list, here per row and compact): col16[row_ptr[i] .. row_ptr[i+1]) holds the
// halo-linear indices q (uint16) of the neighbours of row i.  The pair kernels stage the halo state in shared
// memory in the same order and gather with q.  Positions of halo cells across a periodic seam are shifted by
// -+L when staged, so no minimum-image test is needed in any inner loop.
#pragma once

#include "sph_internal.cuh"

constexpr int kTileMaxHalo = 64;    // (B+2)^d <= 64: B <= 2 in 3D, B <= 6 in 2D
constexpr int kTileMaxTgt = 16;     // B^d <= 16

struct TileTab {                       // one per CTA, in shared memory
    uint32_t h_off[kTileMaxHalo + 1];  // halo-linear offset of each halo cell
    uint32_t h_start[kTileMaxHalo];    // first sorted index of each halo cell
    uint32_t t_off[kTileMaxTgt + 1];   // row offsets of the target cells, in tile-local (z,y,x) order
    int t_cell[kTileMaxTgt];           // halo slot of each target cell
    int ext[3], hs[3], tlo[3], tn[3];  // halo extent, first (unwrapped) halo cell coordinate, slot of the first target, targets
    int nh, nt;
    int seam;                          // some halo cell lies across a periodic face (h_shift != 0)
    uint32_t row0, T, M;               // first sorted row of the tile, rows, halo particles
    float h_shift[3][kTileMaxHalo];    // shift (0, -L or +L per axis) that moves a halo cell next to the tile
};

// Computes the tables of tile `tile`.  Must be called by every thread of the CTA (contains __syncthreads); needs
// at least 2 warps.  Requires ncell >= B+2 on periodic axes (checked on the host).
template <int DIM>
__device__ __forceinline__ void tile_setup(const TileGeom &tg, int tile, const uint32_t *__restrict__ cell_start,
                                           const uint32_t *__restrict__ cell_end, TileTab &tt)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (tg.tabs) {
        // the tables of this tile were written at build time (k_tile_tables): one coalesced read instead of the cell-table
        // look-ups, two scans and three barriers below
        static_assert(sizeof(TileTab) % 4 == 0, "TileTab is copied word by word");
        const uint32_t *src = reinterpret_cast<const uint32_t *>(static_cast<const TileTab *>(tg.tabs) + tile);
        uint32_t *dst = reinterpret_cast<uint32_t *>(&tt);
        for (int i = threadIdx.x; i < (int)(sizeof(TileTab) / 4); i += blockDim.x) dst[i] = __ldg(src + i);
        __syncthreads();
        return;
    }
    if (threadIdx.x == 0) {
        int b = tile, bc[3] = {0, 0, 0};
        bc[0] = b % tg.nb[0];
        b /= tg.nb[0];
        bc[1] = b % tg.nb[1];
        bc[2] = b / tg.nb[1];
        int nh = 1, nt = 1;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            int hs = 0, ext = 1, tlo = 0, tn = 1;
            if (k < DIM) {
                const int c0 = bc[k] * tg.B;
                tn = min(tg.B, tg.ncell[k] - c0);
                if (tg.periodic[k]) {
                    hs = c0 - 1;
                    ext = tn + 2;
                } else {
                    hs = max(c0 - 1, 0);
                    ext = min(c0 + tn, tg.ncell[k] - 1) - hs + 1;
                }
                tlo = c0 - hs;
            }
            tt.hs[k] = hs; tt.ext[k] = ext; tt.tlo[k] = tlo; tt.tn[k] = tn;
            nh *= ext;
            nt *= tn;
        }
        tt.nh = nh;
        tt.nt = nt;
        int seam = 0;
#pragma unroll
        for (int k = 0; k < DIM; ++k)
            if (tg.periodic[k] && (tt.hs[k] < 0 || tt.hs[k] + tt.ext[k] > tg.ncell[k])) seam = 1;
        tt.seam = seam;
    }
    __syncthreads();
    const int nh = tt.nh, nt = tt.nt;
    if (warp == 0) {
        uint32_t c2[2], s2[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int hc = lane * 2 + u;
            c2[u] = 0;
            s2[u] = 0;
            if (hc < nh) {
                int sl[3] = {hc % tt.ext[0], (hc / tt.ext[0]) % tt.ext[1], hc / (tt.ext[0] * tt.ext[1])};
                int64_t lin = 0;
#pragma unroll
                for (int k = DIM - 1; k >= 0; --k) {
                    int c = tt.hs[k] + sl[k];
                    if (tg.periodic[k]) c = c < 0 ? c + tg.ncell[k] : (c >= tg.ncell[k] ? c - tg.ncell[k] : c);
                    lin = lin * tg.ncell[k] + c;
                }
                s2[u] = cell_start[lin];
                c2[u] = cell_end[lin] - s2[u];
                tt.h_start[hc] = s2[u];
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    float sh = 0.f;
                    if (k < DIM && tg.periodic[k]) {
                        const int c = tt.hs[k] + sl[k];
                        sh = c < 0 ? -tg.L[k] : (c >= tg.ncell[k] ? tg.L[k] : 0.f);
                    }
                    tt.h_shift[k][hc] = sh;
                }
            }
        }
        uint32_t tot = c2[0] + c2[1], inc = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        const uint32_t ex = inc - tot;
        if (lane * 2 < nh) tt.h_off[lane * 2] = ex;
        if (lane * 2 + 1 < nh) tt.h_off[lane * 2 + 1] = ex + c2[0];
        if (lane == 31) {
            tt.h_off[nh] = inc;
            tt.M = inc;
        }
    }
    __syncthreads();
    if (warp == 1) {
        // target cells in tile-local (z,y,x) order; rows per target cell; first sorted row of the tile
        uint32_t c = 0, first = 0xffffffffu;
        if (lane < nt) {
            int sl[3] = {lane % tt.tn[0], (lane / tt.tn[0]) % tt.tn[1], lane / (tt.tn[0] * tt.tn[1])};
            const int hc = (tt.tlo[0] + sl[0]) + tt.ext[0] * ((tt.tlo[1] + sl[1]) + tt.ext[1] * (tt.tlo[2] + sl[2]));
            tt.t_cell[lane] = hc;
            c = tt.h_off[hc + 1] - tt.h_off[hc];
            if (c) first = tt.h_start[hc];
        }
        uint32_t inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane < nt) tt.t_off[lane] = inc - c;
        first = __reduce_min_sync(0xffffffffu, first);
        if (lane == 31) {
            tt.t_off[nt] = inc;
            tt.T = inc;
            tt.row0 = inc ? first : 0u;
        }
    }
    __syncthreads();
}

// shift (0 or -+L per axis) that moves the particles of halo cell `hc` next to the tile across a periodic seam
template <int DIM>
__device__ __forceinline__ void tile_cell_shift(const TileGeom &tg, const TileTab &tt, int hc, float sh[3])
{
    sh[0] = tt.h_shift[0][hc];
    sh[1] = tt.h_shift[1][hc];
    sh[2] = DIM == 3 ? tt.h_shift[2][hc] : 0.f;
}

// sorted index of the particle with halo-linear index q (binary search over the <= 64 halo cells)
__device__ __forceinline__ uint32_t tile_q_to_sorted(const TileTab &tt, uint32_t q)
{
    int lo = 0, hi = tt.nh;            // invariant: h_off[lo] <= q < h_off[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (tt.h_off[mid] <= q) lo = mid; else hi = mid;
    }
    return tt.h_start[lo] + (q - tt.h_off[lo]);
}
