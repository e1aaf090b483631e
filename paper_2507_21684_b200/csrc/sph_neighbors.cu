// sph_neighbors.cu -- steps N5-N7 of SURVEY.md 8(a): count / exclusive scan / fill of compact CSR neighbour
// lists (PAPER.md:558 adjacent-cell query; PAPER.md:163 pair list; PAPER.md:167 search radius max{h_i,h_j}),
// plus the export in caller ids.  One warp per row: 32 lanes test 32 candidates of a neighbour cell at a
// time, a ballot compacts the hits, so every row is written coalesced and in a fixed order
// (cells in z,y,x order, ascending sorted index inside a cell) -- deterministic, no atomics.
#include "sph_internal.cuh"

#include <math.h>

namespace {

constexpr int kWarpsPerBlock = 8;

struct SearchPar {
    float scale;     // search_scale (binary32)
    double R;        // scale*hmax*(1+2^-20): half width of the candidate interval per axis
    float band;      // relative half width of the fp32 "too close to call" band
    float Lmax;      // largest periodic box length (0 if none)
};

// R3: the predicate r2 < Hs^2 in binary64 on the wrapped binary32 positions, fixed op order.
__device__ __forceinline__ bool pred_exact(const float4 &a, const float4 &b, float Hs, const GridGeom &gg)
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

// fp32 decision when it is safe (|r2 - Hs^2| outside the rounding band), binary64 sequence otherwise
__device__ __forceinline__ bool pred(const float4 &a, const float4 &b, const SearchPar &sp, const GridGeom &gg,
                                     bool seam)
{
    float Hs = __fmul_rn(sp.scale, fmaxf(a.w, b.w));
    float d0 = a.x - b.x, d1 = a.y - b.y, d2 = gg.dim == 3 ? a.z - b.z : 0.f;
    if (seam) {
        if (gg.periodic[0]) d0 = d0 > 0.5f * gg.L[0] ? d0 - gg.L[0] : (d0 < -0.5f * gg.L[0] ? d0 + gg.L[0] : d0);
        if (gg.periodic[1]) d1 = d1 > 0.5f * gg.L[1] ? d1 - gg.L[1] : (d1 < -0.5f * gg.L[1] ? d1 + gg.L[1] : d1);
        if (gg.dim == 3 && gg.periodic[2])
            d2 = d2 > 0.5f * gg.L[2] ? d2 - gg.L[2] : (d2 < -0.5f * gg.L[2] ? d2 + gg.L[2] : d2);
    }
    float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
    float Hs2 = Hs * Hs;
    float tol = sp.band * (Hs2 + (seam ? Hs * sp.Lmax : 0.f));
    float diff = r2 - Hs2;
    if (fabsf(diff) > tol) return diff < 0.f;
    return pred_exact(a, b, Hs, gg);
}

template <bool FILL>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_neighbors(int64_t n, GridGeom gg, SearchPar sp, const float4 *__restrict__ pos_s,
            const uint32_t *__restrict__ key_sorted, const uint32_t *__restrict__ cell_start,
            const uint32_t *__restrict__ cell_end, uint32_t *__restrict__ cnt,
            const long long *__restrict__ row_ptr, int32_t *__restrict__ col)
{
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
    if (row >= n) return;
    const float4 pi = pos_s[row];
    const float xi[3] = {pi.x, pi.y, pi.z};
    int clo[3] = {0, 0, 0}, chi[3] = {0, 0, 0};
    bool seam = false;
    for (int k = 0; k < gg.dim; ++k) {
        // candidate interval [x - R, x + R]; the cell map is monotone, so every j with |d_k| < Hs lies in it
        int a = cell_coord_raw(__dsub_rn((double)xi[k], sp.R), gg.lo_d[k], gg.edge[k]);
        int b = cell_coord_raw(__dadd_rn((double)xi[k], sp.R), gg.lo_d[k], gg.edge[k]);
        if (gg.periodic[k]) {
            if (b - a + 1 > gg.ncell[k]) b = a + gg.ncell[k] - 1;   // never visit a cell twice
            if (a < 0 || b >= gg.ncell[k]) seam = true;
        } else {
            a = max(a, 0);
            b = min(b, gg.ncell[k] - 1);
        }
        clo[k] = a;
        chi[k] = b;
    }
    uint32_t off = 0;
    const long long base = FILL ? row_ptr[row] : 0;
    for (int cz = clo[2]; cz <= chi[2]; ++cz) {
        int wz = cz;
        if (gg.dim == 3 && gg.periodic[2]) wz = cz < 0 ? cz + gg.ncell[2] : (cz >= gg.ncell[2] ? cz - gg.ncell[2] : cz);
        for (int cy = clo[1]; cy <= chi[1]; ++cy) {
            int wy = cy;
            if (gg.periodic[1]) wy = cy < 0 ? cy + gg.ncell[1] : (cy >= gg.ncell[1] ? cy - gg.ncell[1] : cy);
            for (int cx = clo[0]; cx <= chi[0]; ++cx) {
                int wx = cx;
                if (gg.periodic[0]) wx = cx < 0 ? cx + gg.ncell[0] : (cx >= gg.ncell[0] ? cx - gg.ncell[0] : cx);
                const int64_t lin = wx + (int64_t)gg.ncell[0] * (wy + (int64_t)gg.ncell[1] * wz);
                const uint32_t s = cell_start[lin], e = cell_end[lin];
                for (uint32_t b0 = s; b0 < e; b0 += 32) {
                    const uint32_t j = b0 + lane;
                    bool hit = false;
                    if (j < e) {
                        const float4 pj = pos_s[j];
                        hit = pred(pi, pj, sp, gg, seam);
                    }
                    const uint32_t m = __ballot_sync(0xffffffffu, hit);
                    if (FILL && hit) col[base + off + __popc(m & ((1u << lane) - 1u))] = (int32_t)j;
                    off += __popc(m);
                }
            }
        }
    }
    if (!FILL && lane == 0) cnt[row] = off;
}

// ---------------------------------------------------------------------------------------- export
__global__ void k_export_counts(int64_t n, const uint32_t *__restrict__ inv_perm, const uint32_t *__restrict__ cnt_s,
                                uint32_t *__restrict__ cnt_c)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) cnt_c[i] = cnt_s[inv_perm[i]];
}

// one warp per caller row: translate to caller ids and rank-sort ascending (ids in a row are distinct)
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_export_rows(int64_t n, const uint32_t *__restrict__ inv_perm, const uint32_t *__restrict__ perm,
              const long long *__restrict__ row_ptr_s, const int32_t *__restrict__ col_s,
              const long long *__restrict__ row_ptr_c, int32_t *__restrict__ col_c)
{
    const int lane = threadIdx.x & 31;
    const int64_t i = (int64_t)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
    if (i >= n) return;
    const uint32_t p = inv_perm[i];
    const long long b = row_ptr_s[p], e = row_ptr_s[p + 1], ob = row_ptr_c[i];
    for (long long a = b + lane; a < e; a += 32) {
        const uint32_t id = perm[col_s[a]];
        int rank = 0;
        for (long long c = b; c < e; ++c) rank += perm[col_s[c]] < id ? 1 : 0;
        col_c[ob + rank] = (int32_t)id;
    }
}

} // namespace

extern "C" int sph_neighbors(sph_ctx *ctx, float search_scale, int64_t *nnz_out, sph_stream_t stream)
{
    if (!ctx || !(search_scale >= 1.0f) || !isfinite(search_scale)) return SPH_E_INVALID;
    if (!ctx->cells_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->lists_ready = false;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    const GridGeom &gg = ctx->geom;

    // the statistics of sph_build_cells (error flag, max/min h) are needed on the host to size the search
    uint32_t *hs = reinterpret_cast<uint32_t *>(ctx->h_pinned);
    SPH_CUDA_TRY(cudaMemcpyAsync(hs, ctx->stats.p, 16, cudaMemcpyDeviceToHost, st));
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    if (hs[0] != 0u) return SPH_E_DOMAIN;
    float hmax, hmin;
    memcpy(&hmax, &hs[1], 4);
    memcpy(&hmin, &hs[2], 4);
    ctx->hmax = hmax;
    ctx->hmin = hmin;
    volatile float Rs = search_scale * hmax;
    for (int k = 0; k < gg.dim; ++k)
        if ((double)Rs > gg.edge[k]) return SPH_E_DOMAIN;   // cell_size < search radius

    SearchPar sp;
    sp.scale = search_scale;
    sp.R = (double)Rs * (1.0 + 1.0 / 1048576.0);
    sp.band = 1.0f / 524288.0f;   // 2^-19 relative: > 4x the worst fp32 rounding of r2 (N5)
    sp.Lmax = 0.f;
    for (int k = 0; k < gg.dim; ++k)
        if (gg.periodic[k] && gg.L[k] > sp.Lmax) sp.Lmax = gg.L[k];

    SPH_TRY(ctx->cnt.reserve((size_t)n * 4));
    SPH_TRY(ctx->row_ptr.reserve((size_t)(n + 1) * 8));
    const unsigned nblk = (unsigned)((n + kWarpsPerBlock - 1) / kWarpsPerBlock);
    {
        KScope ks(ctx, SPH_K_COUNT, 1, st);
        k_neighbors<false><<<nblk, kWarpsPerBlock * 32, 0, st>>>(n, gg, sp, ctx->pos_s.as<float4>(),
                                                                ctx->key_sorted.as<uint32_t>(), ctx->cell_start.as<uint32_t>(),
                                                                ctx->cell_end.as<uint32_t>(), ctx->cnt.as<uint32_t>(), nullptr, nullptr);
    }
    {
        KScope ks(ctx, SPH_K_SCAN, 3, st);
        SPH_TRY(sph_scan_u32(ctx, ctx->cnt.as<uint32_t>(), ctx->row_ptr.p, true, n, st));
    }
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->h_pinned + 4, ctx->row_ptr.as<long long>() + n, 8, cudaMemcpyDeviceToHost, st));
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    const int64_t nnz = ctx->h_pinned[4];
    SPH_TRY(ctx->col.reserve((size_t)(nnz > 0 ? nnz : 1) * 4));
    {
        KScope ks(ctx, SPH_K_FILL, 1, st);
        k_neighbors<true><<<nblk, kWarpsPerBlock * 32, 0, st>>>(n, gg, sp, ctx->pos_s.as<float4>(),
                                                               ctx->key_sorted.as<uint32_t>(), ctx->cell_start.as<uint32_t>(),
                                                               ctx->cell_end.as<uint32_t>(), nullptr, ctx->row_ptr.as<long long>(),
                                                               ctx->col.as<int32_t>());
    }
    SPH_CUDA_TRY(cudaGetLastError());
    ctx->nnz = nnz;
    ctx->search_scale = search_scale;
    ctx->lists_ready = true;
    if (nnz_out) *nnz_out = nnz;
    return SPH_OK;
}

extern "C" int sph_neighbors_export(sph_ctx *ctx, int64_t *row_ptr, int32_t *col_idx, sph_stream_t stream)
{
    if (!ctx || !row_ptr || !col_idx) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    SPH_TRY(ctx->s3.reserve((size_t)n * 4));
    uint32_t *cnt_c = ctx->s3.as<uint32_t>();
    KScope ks(ctx, SPH_K_EXPORT, 5, st);
    k_export_counts<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, ctx->inv_perm.as<uint32_t>(), ctx->cnt.as<uint32_t>(), cnt_c);
    SPH_TRY(sph_scan_u32(ctx, cnt_c, row_ptr, true, n, st));
    k_export_rows<<<(unsigned)((n + kWarpsPerBlock - 1) / kWarpsPerBlock), kWarpsPerBlock * 32, 0, st>>>(
        n, ctx->inv_perm.as<uint32_t>(), ctx->perm.as<uint32_t>(), ctx->row_ptr.as<long long>(), ctx->col.as<int32_t>(),
        (const long long *)row_ptr, col_idx);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}
