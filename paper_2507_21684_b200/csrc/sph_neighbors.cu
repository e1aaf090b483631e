// sph_neighbors.cu -- steps N5-N7 of SURVEY.md 8(a): count / exclusive scan / fill of compact CSR neighbour
// lists (PAPER.md:558 adjacent-cell query; PAPER.md:163 pair list; PAPER.md:167 search radius max{h_i,h_j}),
// plus the export in caller ids.  One warp per row: 32 lanes test 32 candidates of a neighbour cell at a
// time, a ballot compacts the hits, so every row is written coalesced and in a fixed order
// (cells in z,y,x order, ascending sorted index inside a cell) -- deterministic, no atomics.
#include "sph_internal.cuh"
#include "sph_tiles.cuh"
#include "sph_search.cuh"

#include <math.h>

namespace {

constexpr int kWarpsPerBlock = 8;

// ---------------------------------------------------------------------------------------- tile search
// One CTA owns a block of B^d cells.  It stages the particles of the (B+2)^d halo cells into shared memory
// (contiguous runs of the cell-sorted array; positions pre-shifted by +-L across a periodic seam, so the inner
// loop needs no minimum image), then one warp per target row scans the 3^(d-1) x-runs of 3 adjacent cells that
// make up the row's 3^d neighbour cells: 32 candidates per iteration from shared memory, ballot compaction.
// The halo is processed in chunks of `cap` candidates, so any cell occupancy works; a block whose halo fits one
// chunk (the normal case) keeps all row state in registers.
struct TilePar {
    int B;             // block edge in cells
    int nb[3];         // blocks per axis
    int cap;           // candidates per shared-memory chunk
    int slow[3];       // periodic axis with fewer than B+2 cells: halo = all cells, minimum image in the loop
};

constexpr int kMaxHalo = 64;     // (B+2)^d <= 64: B = 2 in 3D, B <= 6 in 2D

template <int DIM, bool FILL>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_neighbors_tile(int64_t n, GridGeom gg, SearchPar sp, TilePar tp, const float4 *__restrict__ pos_s,
                 const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
                 uint32_t *__restrict__ cnt, uint32_t *__restrict__ cursor, const long long *__restrict__ row_ptr,
                 int32_t *__restrict__ col)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *cand = reinterpret_cast<float4 *>(smem_raw);
    uint32_t *gidx = reinterpret_cast<uint32_t *>(smem_raw + (size_t)tp.cap * sizeof(float4));
    __shared__ uint32_t h_off[kMaxHalo + 1];      // halo-linear offset of each halo cell
    __shared__ uint32_t h_start[kMaxHalo];        // first sorted index of each halo cell
    __shared__ uint32_t t_off[kMaxHalo + 1];      // target-row offsets (targets are halo cells too)
    __shared__ int t_cell[kMaxHalo];              // halo cell id of each target cell

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int bc[3] = {0, 0, 0};
    {
        int b = blockIdx.x;
        bc[0] = b % tp.nb[0];
        b /= tp.nb[0];
        bc[1] = b % tp.nb[1];
        bc[2] = b / tp.nb[1];
    }
    // halo extent per axis: hs = first (unwrapped) cell coordinate, ext = number of cells, tlo = slot of the first target
    int hs[3] = {0, 0, 0}, ext[3] = {1, 1, 1}, tlo[3] = {0, 0, 0}, tn[3] = {1, 1, 1};
    bool seam = false;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        const int c0 = bc[k] * tp.B;
        tn[k] = min(tp.B, gg.ncell[k] - c0);
        if (gg.periodic[k]) {
            if (tp.slow[k]) {
                hs[k] = 0;
                ext[k] = gg.ncell[k];
                seam = true;
            } else {
                hs[k] = c0 - 1;
                ext[k] = tn[k] + 2;
                if (hs[k] < 0 || hs[k] + ext[k] > gg.ncell[k]) seam = true;
            }
        } else {
            hs[k] = max(c0 - 1, 0);
            ext[k] = min(c0 + tn[k], gg.ncell[k] - 1) - hs[k] + 1;
        }
        tlo[k] = c0 - hs[k];
    }
    const int nh = ext[0] * ext[1] * ext[2];
    const int nt = tn[0] * tn[1] * tn[2];

    // ---- halo tables (warp 0: two cells per lane, warp scan)
    if (warp == 0) {
        uint32_t c2[2], s2[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int hc = lane * 2 + u;
            c2[u] = 0;
            s2[u] = 0;
            if (hc < nh) {
                int sl[3] = {hc % ext[0], (hc / ext[0]) % ext[1], hc / (ext[0] * ext[1])};
                int64_t lin = 0;
#pragma unroll
                for (int k = DIM - 1; k >= 0; --k) {
                    int c = hs[k] + sl[k];
                    if (gg.periodic[k]) c = c < 0 ? c + gg.ncell[k] : (c >= gg.ncell[k] ? c - gg.ncell[k] : c);
                    lin = lin * gg.ncell[k] + c;
                }
                s2[u] = cell_start[lin];
                c2[u] = cell_end[lin] - s2[u];
                h_start[hc] = s2[u];
            }
        }
        uint32_t tot = c2[0] + c2[1], inc = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        const uint32_t ex = inc - tot;
        if (lane * 2 < nh) h_off[lane * 2] = ex;
        if (lane * 2 + 1 < nh) h_off[lane * 2 + 1] = ex + c2[0];
        if (lane == 31) h_off[nh] = inc;
    }
    __syncthreads();
    if (warp == 1) {
        // target cells in (z,y,x) order = ascending halo cell id; rows per target cell
        uint32_t c2[2] = {0, 0};
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int tc = lane * 2 + u;
            if (tc < nt) {
                int sl[3] = {tc % tn[0], (tc / tn[0]) % tn[1], tc / (tn[0] * tn[1])};
                const int hc = (tlo[0] + sl[0]) + ext[0] * ((tlo[1] + sl[1]) + ext[1] * (tlo[2] + sl[2]));
                t_cell[tc] = hc;
                c2[u] = h_off[hc + 1] - h_off[hc];
            }
        }
        uint32_t tot = c2[0] + c2[1], inc = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        const uint32_t ex = inc - tot;
        if (lane * 2 < nt) t_off[lane * 2] = ex;
        if (lane * 2 + 1 < nt) t_off[lane * 2 + 1] = ex + c2[0];
        if (lane == 31) t_off[nt] = inc;
    }
    __syncthreads();
    const uint32_t M = h_off[nh], T = t_off[nt];
    if (T == 0) return;
    const bool single = M <= (uint32_t)tp.cap;
    const float tol_rel = sp.band;

    for (uint32_t c0 = 0; c0 < M; c0 += (uint32_t)tp.cap) {
        const uint32_t c1 = min(M, c0 + (uint32_t)tp.cap);
        if (c0 > 0) __syncthreads();
        // ---- stage the chunk [c0, c1) of the halo-linear candidate sequence
        for (int hc = warp; hc < nh; hc += kWarpsPerBlock) {
            const uint32_t o0 = h_off[hc], o1 = h_off[hc + 1];
            if (o1 <= c0 || o0 >= c1) continue;
            float sh[3] = {0.f, 0.f, 0.f};
            {
                int sl[3] = {hc % ext[0], (hc / ext[0]) % ext[1], hc / (ext[0] * ext[1])};
#pragma unroll
                for (int k = 0; k < DIM; ++k)
                    if (gg.periodic[k] && !tp.slow[k]) {
                        const int c = hs[k] + sl[k];
                        sh[k] = c < 0 ? -gg.L[k] : (c >= gg.ncell[k] ? gg.L[k] : 0.f);
                    }
            }
            const uint32_t gs = h_start[hc];
            for (uint32_t q = max(o0, c0) + lane; q < min(o1, c1); q += 32) {
                const uint32_t g = gs + (q - o0);
                float4 pj = pos_s[g];
                pj.x += sh[0];
                pj.y += sh[1];
                if (DIM == 3) pj.z += sh[2];
                cand[q - c0] = pj;
                gidx[q - c0] = g;
            }
        }
        __syncthreads();
        // ---- rows: one warp per target row
        for (uint32_t t = warp; t < T; t += kWarpsPerBlock) {
            int tc = 0;
            while (t >= t_off[tc + 1]) ++tc;
            const int hc_i = t_cell[tc];
            const uint32_t row = h_start[hc_i] + (t - t_off[tc]);
            const float4 pi = pos_s[row];
            int sl[3] = {hc_i % ext[0], (hc_i / ext[0]) % ext[1], hc_i / (ext[0] * ext[1])};
            uint32_t off = 0;
            if (!single && c0 > 0) off = FILL ? cursor[row] : cnt[row];
            const long long base = FILL ? row_ptr[row] : 0;
            // neighbour cells of the row: dz, dy in {-1,0,1}; along x either one merged run or cell by cell
            const int zlo = DIM == 3 ? -1 : 0, zhi = DIM == 3 ? 1 : 0;
            for (int dz = zlo; dz <= zhi; ++dz) {
                int sz = sl[2] + dz;
                if (DIM == 3) {
                    if (tp.slow[2]) sz = sz < 0 ? sz + ext[2] : (sz >= ext[2] ? sz - ext[2] : sz);
                    else if (sz < 0 || sz >= ext[2]) continue;
                }
                for (int dy = -1; dy <= 1; ++dy) {
                    int sy = sl[1] + dy;
                    if (tp.slow[1]) sy = sy < 0 ? sy + ext[1] : (sy >= ext[1] ? sy - ext[1] : sy);
                    else if (sy < 0 || sy >= ext[1]) continue;
                    const int rowbase = ext[0] * (sy + ext[1] * sz);
                    const int nrun = tp.slow[0] ? 3 : 1;
                    for (int rr = 0; rr < nrun; ++rr) {
                        int xa, xb;                       // first / last halo slot along x of this run
                        if (tp.slow[0]) {
                            int sx = sl[0] + rr - 1;
                            sx = sx < 0 ? sx + ext[0] : (sx >= ext[0] ? sx - ext[0] : sx);
                            xa = xb = sx;
                        } else {
                            xa = max(sl[0] - 1, 0);
                            xb = min(sl[0] + 1, ext[0] - 1);
                        }
                        uint32_t q0 = max(h_off[rowbase + xa], c0), q1 = min(h_off[rowbase + xb + 1], c1);
                        for (uint32_t qb = q0; qb < q1; qb += 32) {
                            const uint32_t q = qb + lane;
                            bool hit = false;
                            uint32_t g = 0;
                            if (q < q1) {
                                const float4 pj = cand[q - c0];
                                const float Hs = __fmul_rn(sp.scale, fmaxf(pi.w, pj.w));
                                float d0 = pi.x - pj.x, d1 = pi.y - pj.y, d2 = DIM == 3 ? pi.z - pj.z : 0.f;
                                if (tp.slow[0]) d0 = d0 > 0.5f * gg.L[0] ? d0 - gg.L[0] : (d0 < -0.5f * gg.L[0] ? d0 + gg.L[0] : d0);
                                if (tp.slow[1]) d1 = d1 > 0.5f * gg.L[1] ? d1 - gg.L[1] : (d1 < -0.5f * gg.L[1] ? d1 + gg.L[1] : d1);
                                if (DIM == 3 && tp.slow[2])
                                    d2 = d2 > 0.5f * gg.L[2] ? d2 - gg.L[2] : (d2 < -0.5f * gg.L[2] ? d2 + gg.L[2] : d2);
                                const float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
                                const float Hs2 = Hs * Hs;
                                const float tol = tol_rel * (seam ? fmaf(Hs, sp.Lmax, Hs2) : Hs2);
                                const float diff = r2 - Hs2;
                                hit = diff < 0.f;
                                g = gidx[q - c0];
                                if (fabsf(diff) <= tol) hit = pred_exact(pi, pos_s[g], Hs, gg);   // R3, binary64
                            }
                            const uint32_t m = __ballot_sync(0xffffffffu, hit);
                            if (FILL && hit) col[base + off + __popc(m & ((1u << lane) - 1u))] = (int32_t)g;
                            off += __popc(m);
                        }
                    }
                }
            }
            if (lane == 0) {
                if (FILL) {
                    if (!single) cursor[row] = off;
                } else {
                    cnt[row] = off;
                }
            }
        }
    }
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

    // candidate cell-block decompositions: their largest halo decides whether the tile-local layout fits
    int cand[3], ncand = 0;
    if (ctx->opt_list_mode != 1) ncand = sph_tile_candidates(ctx, cand);
    if (ncand) SPH_TRY(sph_tile_stats_launch(ctx, cand, ncand, st));
    const bool fused_stats = ncand && ctx->opt_build_fused;
    if (fused_stats) {
        SPH_TRY(sph_fused_stats_launch(ctx, st));
        SPH_CUDA_TRY(cudaMemcpyAsync(ctx->h_pinned + 16, ctx->fstats.p, 16, cudaMemcpyDeviceToHost, st));
    }
    // the statistics of sph_build_cells (error flag, max/min h) are needed on the host to size the search
    uint32_t hs[16];
    uint32_t *hpin = reinterpret_cast<uint32_t *>(ctx->h_pinned + 8);
    SPH_CUDA_TRY(cudaMemcpyAsync(hpin, ctx->stats.p, 64, cudaMemcpyDeviceToHost, st));
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    memcpy(hs, hpin, 64);
    ctx->f_ncmax = 0;
    ctx->f_pairs = 0;
    if (fused_stats) {
        memcpy(&ctx->f_ncmax, ctx->h_pinned + 16, 4);
        memcpy(&ctx->f_pairs, ctx->h_pinned + 17, 8);
    }
    if (hs[0] != 0u) return SPH_E_DOMAIN;
    float hmax, hmin;
    memcpy(&hmax, &hs[1], 4);
    memcpy(&hmin, &hs[2], 4);
    ctx->hmax = hmax;
    ctx->hmin = hmin;
    if (ctx->scale_slack_cap > 0.f && hmax > 0.f) {
        // sph_rk_step (automatic Verlet skin): take the slack the cell size leaves, up to the cap; the product
        // scale * hmax must stay <= every cell edge in binary32, as the check below demands
        double emin = gg.edge[0];
        for (int k = 1; k < gg.dim; ++k) emin = gg.edge[k] < emin ? gg.edge[k] : emin;
        float s = (float)(emin / (double)hmax);
        for (int it = 0; it < 4; ++it) {
            volatile float prod = s * hmax;
            if ((double)prod <= emin) break;
            s = nextafterf(s, 0.f);
        }
        s = fminf(s, search_scale + ctx->scale_slack_cap);
        if (s >= search_scale + 0.02f) search_scale = s;     // less than that is not worth a longer list
    }
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
    sp.Hs_u = Rs;                                   // = (float)(scale*h) when h is uniform

    ctx->tile_mode = false;
    ctx->col_valid = false;
    for (int k = 0; k < ncand; ++k) {
        const uint32_t Mmax = hs[4 + 2 * k], Tmax = hs[5 + 2 * k];
        if (!sph_tile_fits(gg.dim, Mmax)) continue;
        SPH_TRY(sph_neighbors_tile_run(ctx, sp, cand[k], Mmax, Tmax, hs[10], st, nnz_out));
        ctx->tile_Mhalf = (gg.dim == 3 && cand[k] == 2) ? hs[kTileHalfSlot] : 0u;
        ctx->search_scale = search_scale;
        ctx->lists_ready = true;
        return SPH_OK;
    }
    // no halo fits the pair kernels: the tile SEARCH (positions only) may still fit; its lists are translated to
    // sorted ids and the generic pair kernels run on them
    if (ctx->opt_list_mode == 0)
        for (int k = ncand - 1; k >= 0; --k) {
            const uint32_t Mmax = hs[4 + 2 * k], Tmax = hs[5 + 2 * k];
            if (!sph_tile_search_fits(Mmax)) continue;
            SPH_TRY(sph_neighbors_tile_run(ctx, sp, cand[k], Mmax, Tmax, hs[10], st, nnz_out));
            SPH_TRY(sph_tile_expand_col(ctx, st));
            ctx->tile_mode = false;
            ctx->search_scale = search_scale;
            ctx->lists_ready = true;
            return SPH_OK;
        }

    SPH_TRY(ctx->cnt.reserve((size_t)n * 4));
    SPH_TRY(ctx->row_ptr.reserve((size_t)(n + 1) * 8));
    // tile geometry: block edge B and chunk capacity from the mean cell occupancy (any occupancy is handled
    // by chunking; this only picks the fast configuration)
    TilePar tp;
    memset(&tp, 0, sizeof(tp));
    const double mean_occ = (double)n / (double)ctx->ncells_total;
    const int cap_max = 8192;                                       // 160 KB of shared memory
    if (gg.dim == 3) tp.B = 64.0 * mean_occ * 1.25 <= cap_max ? 2 : 1;
    else tp.B = 36.0 * mean_occ * 1.25 <= cap_max ? 4 : (16.0 * mean_occ * 1.25 <= cap_max ? 2 : 1);
    double halo_cells = 1.0;
    int64_t nblocks = 1;
    for (int k = 0; k < 3; ++k) {
        tp.nb[k] = 1;
        if (k < gg.dim) {
            tp.nb[k] = (gg.ncell[k] + tp.B - 1) / tp.B;
            tp.slow[k] = gg.periodic[k] && gg.ncell[k] < tp.B + 2;
            halo_cells *= tp.slow[k] ? gg.ncell[k] : tp.B + 2;
        }
        nblocks *= tp.nb[k];
    }
    {
        double want = halo_cells * mean_occ * 1.25 + 64.0;
        int cap = (int)((want + 255.0) / 256.0) * 256;
        tp.cap = cap < 1024 ? 1024 : (cap > cap_max ? cap_max : cap);
    }
    const size_t smem = (size_t)tp.cap * (sizeof(float4) + sizeof(uint32_t));
    SPH_TRY(ctx->s3.reserve((size_t)n * 4));                        // cursor of the multi-chunk fill path
    uint32_t *cursor = ctx->s3.as<uint32_t>();
#define SPH_NB_LAUNCH(DIM, FILL, CNT, RP, COL)                                                                        \
    do {                                                                                                              \
        SPH_CUDA_TRY(cudaFuncSetAttribute(k_neighbors_tile<DIM, FILL>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                                          (int)smem));                                                                \
        k_neighbors_tile<DIM, FILL><<<(unsigned)nblocks, kWarpsPerBlock * 32, smem, st>>>(                            \
            n, gg, sp, tp, ctx->pos_s.as<float4>(), ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), CNT, \
            cursor, RP, COL);                                                                                         \
    } while (0)
    {
        KScope ks(ctx, SPH_K_COUNT, 1, st);
        if (gg.dim == 3) SPH_NB_LAUNCH(3, false, ctx->cnt.as<uint32_t>(), nullptr, nullptr);
        else SPH_NB_LAUNCH(2, false, ctx->cnt.as<uint32_t>(), nullptr, nullptr);
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
        if (gg.dim == 3) SPH_NB_LAUNCH(3, true, nullptr, ctx->row_ptr.as<long long>(), ctx->col.as<int32_t>());
        else SPH_NB_LAUNCH(2, true, nullptr, ctx->row_ptr.as<long long>(), ctx->col.as<int32_t>());
    }
#undef SPH_NB_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    ctx->nnz = nnz;
    ctx->col_valid = true;
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
    SPH_TRY(sph_tile_expand_col(ctx, st));
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
