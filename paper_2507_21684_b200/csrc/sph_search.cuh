// sph_search.cuh -- parameters and the exact predicate of the neighbour search (reading R3 of DESIGN.md),
// shared by the generic search (sph_neighbors.cu) and the tile search (sph_neighbors_tile.cu).
#pragma once

#include "sph_internal.cuh"

struct SearchPar {
    float scale;     // search_scale (binary32)
    double R;        // scale*hmax*(1+2^-20): half width of the candidate interval per axis
    float band;      // relative half width of the fp32 "too close to call" band
    float Lmax;      // largest periodic box length (0 if none)
    float Hs_u;      // (float)(scale*h) when h is uniform
};

// R3: the predicate r2 < Hs^2 in binary64 on the wrapped binary32 positions, fixed op order.
static __device__ __forceinline__ bool pred_exact(const float4 &a, const float4 &b, float Hs, const GridGeom &gg)
{
    double d0 = __dsub_rn((double)a.x, (double)b.x);
    double d1 = __dsub_rn((double)a.y, (double)b.y);
    double d2 = gg.dim == 3 ? __dsub_rn((double)a.z, (double)b.z) : 0.0;
    if (gg.periodic[0]) {
        double L = gg.L_d[0];
        if (d0 > 0.5 * L) d0 = __dsub_rn(d0, L);
        else if (d0 < -0.5 * L) d0 = __dadd_rn(d0, L);
    }
    if (gg.periodic[1]) {
        double L = gg.L_d[1];
        if (d1 > 0.5 * L) d1 = __dsub_rn(d1, L);
        else if (d1 < -0.5 * L) d1 = __dadd_rn(d1, L);
    }
    if (gg.dim == 3 && gg.periodic[2]) {
        double L = gg.L_d[2];
        if (d2 > 0.5 * L) d2 = __dsub_rn(d2, L);
        else if (d2 < -0.5 * L) d2 = __dadd_rn(d2, L);
    }
    double r2 = __dmul_rn(d0, d0);
    r2 = __fma_rn(d1, d1, r2);
    if (gg.dim == 3) r2 = __fma_rn(d2, d2, r2);
    double Hs2 = __dmul_rn((double)Hs, (double)Hs);
    return r2 < Hs2;
}


// tile search (sph_neighbors_tile.cu)
int sph_tile_candidates(const sph_ctx *ctx, int out[3]);
int sph_tile_stats_launch(sph_ctx *ctx, const int *cand, int ncand, cudaStream_t st);
bool sph_tile_fits(int dim, uint32_t Mmax);
bool sph_tile_search_fits(uint32_t Mmax);
int sph_neighbors_tile_run(sph_ctx *ctx, const SearchPar &sp, int B, uint32_t Mmax, uint32_t Tmax, uint32_t occmax,
                           cudaStream_t st, int64_t *nnz_out);
