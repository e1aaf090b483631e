// sph_cells.cu -- steps N1-N4 of SURVEY.md 8(a): wrap + Morton cell key, stable LSD radix sort,
// reorder into sorted float4 SoA, cell start/end table; plus the device-wide exclusive scan used by N6.
// Hand-written for sm_100a; no library sort/scan.  PAPER.md:556-560 (cells, compact map, space-filling curve).
#include "sph_internal.cuh"

#include <math.h>

#include <mutex>

namespace {

constexpr int kThreads = 256;

// ------------------------------------------------------------------------------------------ N1
// wrap (R4), cell coordinate (binary64, monotone), Morton key; error flag; min/max of h.
// stats[0] = error bits (1: position outside a bounded axis or non-finite, 2: h non-finite or <= 0),
// stats[1] = max h (float bits), stats[2] = min h (float bits)   -- integer atomics only.
__global__ void k_wrap_key(const float *__restrict__ x, const float *__restrict__ h, int64_t n, GridGeom gg,
                           uint32_t *__restrict__ key, uint32_t *__restrict__ stats)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t err = 0;
    float hv = 0.f;
    bool live = i < n;
    if (live) {
        int c[3] = {0, 0, 0};
        for (int k = 0; k < gg.dim; ++k) {
            float xv = x[i * gg.dim + k];
            if (!isfinite(xv)) {
                err |= 1u;
                continue;
            }
            float w = xv;
            if (gg.periodic[k])
                w = wrap_coord(xv, gg.lo[k], gg.hi[k], gg.L[k]);
            else if (xv < gg.lo[k] || xv >= gg.hi[k])
                err |= 1u;
            int cc = cell_coord_raw((double)w, gg.lo_d[k], gg.edge[k]);
            cc = max(0, min(gg.ncell[k] - 1, cc));
            c[k] = cc;
        }
        key[i] = morton_encode(gg.dim, c[0], c[1], c[2]);
        hv = h[i];
        if (!isfinite(hv) || !(hv > 0.f)) {
            err |= 2u;
            hv = 0.f;
        }
    }
    // warp-aggregate the statistics, one atomic per warp
    uint32_t hb = __float_as_uint(hv);
    uint32_t hmaxb = __reduce_max_sync(0xffffffffu, hb);
    uint32_t hminb = __reduce_min_sync(0xffffffffu, live && hv > 0.f ? hb : 0x7f7fffffu);
    uint32_t e = __reduce_or_sync(0xffffffffu, err);
    if ((threadIdx.x & 31) == 0) {
        // same-address atomics serialise in L2 (65 k warps x 3 atomics cost ~80 us here): only a warp that can still
        // change the statistic issues one; the plain read may be stale, which only costs a redundant atomic
        const volatile uint32_t *vs = stats;
        if (e) atomicOr(&stats[0], e);
        if (hmaxb > vs[1]) atomicMax(&stats[1], hmaxb);
        if (hminb < vs[2]) atomicMin(&stats[2], hminb);
    }
}

// ------------------------------------------------------------------------------------------ N2
// Stable LSD radix sort, digits of up to kRsMaxBits bits (the host picks the fewest passes that cover the key, then the
// narrowest digit for that many passes).  Each warp owns a contiguous chunk of kChunk keys and ranks them
// round by round (32 keys per round) with __match_any_sync, so equal keys keep their input order.
constexpr int kRsWarps = 8;
constexpr int kRsItems = 16;
constexpr int kChunk = 32 * kRsItems;
constexpr int kRsMaxBits = 9;
constexpr int kRsMaxBins = 1 << kRsMaxBits;

__global__ void __launch_bounds__(kRsWarps * 32)
k_radix_hist(const uint32_t *__restrict__ key, int64_t n, int shift, int bits, int64_t nchunks, uint32_t *__restrict__ hist)
{
    __shared__ uint32_t cnt[kRsWarps][kRsMaxBins];
    const uint32_t bins = 1u << bits, mask = bins - 1u;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t chunk = (int64_t)blockIdx.x * kRsWarps + warp;
    for (uint32_t d = lane; d < bins; d += 32) cnt[warp][d] = 0;
    __syncwarp();
    if (chunk < nchunks) {
        const int64_t base = chunk * kChunk;
        for (int r = 0; r < kRsItems; ++r) {
            int64_t i = base + r * 32 + lane;
            uint32_t d = i < n ? ((key[i] >> shift) & mask) : bins;
            uint32_t peers = __match_any_sync(0xffffffffu, d);
            if (d < bins && (peers & ((1u << lane) - 1u)) == 0u) cnt[warp][d] += __popc(peers);
            __syncwarp();
        }
        for (uint32_t d = lane; d < bins; d += 32) hist[(int64_t)d * nchunks + chunk] = cnt[warp][d];
    }
}

__global__ void __launch_bounds__(kRsWarps * 32)
k_radix_scatter(const uint32_t *__restrict__ key_in, const uint32_t *__restrict__ val_in,
                uint32_t *__restrict__ key_out, uint32_t *__restrict__ val_out, int64_t n, int shift, int bits,
                int64_t nchunks, const uint32_t *__restrict__ hist_scanned)
{
    __shared__ uint32_t off[kRsWarps][kRsMaxBins];
    const uint32_t bins = 1u << bits, mask = bins - 1u;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t chunk = (int64_t)blockIdx.x * kRsWarps + warp;
    if (chunk >= nchunks) return;
    for (uint32_t d = lane; d < bins; d += 32) off[warp][d] = hist_scanned[(int64_t)d * nchunks + chunk];
    __syncwarp();
    const int64_t base = chunk * kChunk;
    for (int r = 0; r < kRsItems; ++r) {
        int64_t i = base + r * 32 + lane;
        bool live = i < n;
        uint32_t k = live ? key_in[i] : 0u;
        uint32_t v = live ? (val_in ? val_in[i] : (uint32_t)i) : 0u;
        uint32_t d = live ? ((k >> shift) & mask) : bins;
        uint32_t peers = __match_any_sync(0xffffffffu, d);
        uint32_t lower = peers & ((1u << lane) - 1u);
        uint32_t pos = 0;
        if (live) pos = off[warp][d] + __popc(lower);
        __syncwarp();
        if (live && lower == 0u) off[warp][d] += __popc(peers);
        __syncwarp();
        if (live) {
            key_out[pos] = k;
            val_out[pos] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------ scan
constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ unsigned long long block_exclusive_scan(unsigned long long v, unsigned long long *total)
{
    __shared__ unsigned long long wsum[kScanThreads / 32];
    __shared__ unsigned long long tot;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        unsigned long long w = lane < kScanThreads / 32 ? wsum[lane] : 0ull;
        unsigned long long winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        if (lane < kScanThreads / 32) wsum[lane] = winc - w;
        if (lane == kScanThreads / 32 - 1) tot = winc;
    }
    __syncthreads();
    unsigned long long r = inc - v + wsum[warp];
    *total = tot;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_reduce(const uint32_t *__restrict__ in, int64_t m, unsigned long long *__restrict__ block_sums)
{
    const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < m) s += in[base + k];
    unsigned long long tot;
    block_exclusive_scan(s, &tot);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = tot;
}

// single block: exclusive scan of the block sums, sequential over tiles of kScanThreads with a carry
__global__ void __launch_bounds__(kScanThreads)
k_scan_sums(unsigned long long *__restrict__ block_sums, int64_t nb)
{
    unsigned long long carry = 0;
    for (int64_t base = 0; base < nb; base += kScanThreads) {
        int64_t i = base + threadIdx.x;
        unsigned long long v = i < nb ? block_sums[i] : 0ull;
        unsigned long long tot;
        unsigned long long ex = block_exclusive_scan(v, &tot);
        if (i < nb) block_sums[i] = ex + carry;
        carry += tot;
    }
}

template <class OutT>
__global__ void __launch_bounds__(kScanThreads)
k_scan_apply(const uint32_t *__restrict__ in, OutT *__restrict__ out, int64_t m,
             const unsigned long long *__restrict__ block_sums, int write_total)
{
    const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = base + k < m ? in[base + k] : 0u;
        s += v[k];
    }
    unsigned long long tot;
    unsigned long long ex = block_exclusive_scan(s, &tot) + block_sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < m) out[base + k] = (OutT)ex;
        ex += v[k];
    }
    if (write_total && blockIdx.x == gridDim.x - 1 && threadIdx.x == kScanThreads - 1) out[m] = (OutT)ex;
}

// ------------------------------------------------------------------------------------------ N3 + N4
// gather the caller's data into sorted order; mark cell boundaries (head flags of the sorted key run)
__global__ void k_reorder(const float *__restrict__ x, const float *__restrict__ h, int64_t n, GridGeom gg,
                          const uint32_t *__restrict__ key_sorted, const uint32_t *__restrict__ idx_sorted,
                          uint32_t *__restrict__ perm, uint32_t *__restrict__ inv_perm, float4 *__restrict__ pos_s,
                          uint32_t *__restrict__ cell_start, uint32_t *__restrict__ cell_end)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    uint32_t i = idx_sorted[p];
    perm[p] = i;
    inv_perm[i] = (uint32_t)p;
    float w[3] = {0.f, 0.f, 0.f};
    for (int k = 0; k < gg.dim; ++k) {
        float xv = x[(int64_t)i * gg.dim + k];
        w[k] = gg.periodic[k] && isfinite(xv) ? wrap_coord(xv, gg.lo[k], gg.hi[k], gg.L[k]) : xv;
    }
    pos_s[p] = make_float4(w[0], w[1], w[2], h[i]);
    uint32_t kc = key_sorted[p];
    int cx, cy, cz;
    morton_decode(gg.dim, kc, cx, cy, cz);
    int64_t lin = cx + (int64_t)gg.ncell[0] * (cy + (int64_t)gg.ncell[1] * cz);
    if (p == 0 || key_sorted[p - 1] != kc) cell_start[lin] = (uint32_t)p;
    if (p == n - 1 || key_sorted[p + 1] != kc) cell_end[lin] = (uint32_t)(p + 1);
}

// ------------------------------------------------------------------------------------------ Verlet validity
// largest minimum-image displacement since the build; float bits of a non-negative float order like
// unsigned integers, so the maximum is an integer atomic
__global__ void k_max_displacement(const float *__restrict__ x, const float *__restrict__ h, int64_t n, GridGeom gg,
                                   const uint32_t *__restrict__ inv_perm, const float4 *__restrict__ pos_s,
                                   uint32_t *__restrict__ out)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    float r = 0.f;
    if (i < n) {
        const float4 b = pos_s[inv_perm[i]];
        const float xb[3] = {b.x, b.y, b.z};
        float r2 = 0.f;
        bool outside = false;
        for (int k = 0; k < gg.dim; ++k) {
            float xv = x[i * gg.dim + k];
            float d;
            if (gg.periodic[k]) {
                d = wrap_coord(xv, gg.lo[k], gg.hi[k], gg.L[k]) - xb[k];
                d = d > 0.5f * gg.L[k] ? d - gg.L[k] : (d < -0.5f * gg.L[k] ? d + gg.L[k] : d);
            } else {
                d = xv - xb[k];
                if (!(xv >= gg.lo[k] && xv <= gg.hi[k])) outside = true;
            }
            r2 = fmaf(d, d, r2);
        }
        r = sqrtf(r2);
        // left a bounded axis: never valid, so the caller rebuilds and sph_build_cells reports SPH_E_DOMAIN
        if (outside) r = __uint_as_float(0x7f800000u);
        if (!(r >= 0.f)) r = __uint_as_float(0x7f800000u);        // NaN position: never valid
        if (h && h[i] != b.w) r = __uint_as_float(0x7f800000u);   // the lists were built for another h: never valid
    }
    uint32_t rb = __reduce_max_sync(0xffffffffu, __float_as_uint(r));
    if ((threadIdx.x & 31) == 0 && rb > *(volatile uint32_t *)out) atomicMax(out, rb);
}

int ceil_log2(int v)
{
    int b = 0;
    while ((1 << b) < v) ++b;
    return b;
}

} // namespace

// exclusive scan of m uint32 values; out is uint32[m] or (out64) int64[m+1] with the total at out[m]
int sph_scan_u32(sph_ctx *ctx, const uint32_t *in, void *out, bool out64, int64_t m, cudaStream_t st)
{
    if (m <= 0) return SPH_OK;
    int64_t nb = (m + kScanTile - 1) / kScanTile;
    SPH_TRY(ctx->scan_tmp.reserve((size_t)nb * sizeof(unsigned long long)));
    auto *sums = ctx->scan_tmp.as<unsigned long long>();
    k_scan_reduce<<<(unsigned)nb, kScanThreads, 0, st>>>(in, m, sums);
    k_scan_sums<<<1, kScanThreads, 0, st>>>(sums, nb);
    if (out64)
        k_scan_apply<long long><<<(unsigned)nb, kScanThreads, 0, st>>>(in, (long long *)out, m, sums, 1);
    else
        k_scan_apply<uint32_t><<<(unsigned)nb, kScanThreads, 0, st>>>(in, (uint32_t *)out, m, sums, 0);
    // three launches; counted by the caller's KScope
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

static int make_geom(const sph_domain *dom, GridGeom *gg, int64_t *ncells_total)
{
    if (dom->dim != 2 && dom->dim != 3) return SPH_E_INVALID;
    if (!(dom->cell_size > 0.f) || !isfinite(dom->cell_size)) return SPH_E_DOMAIN;
    memset(gg, 0, sizeof(*gg));
    gg->dim = dom->dim;
    int maxnc = 1;
    int64_t tot = 1;
    for (int k = 0; k < 3; ++k) {
        gg->ncell[k] = 1;
        gg->edge[k] = 1.0;
    }
    for (int k = 0; k < dom->dim; ++k) {
        gg->periodic[k] = dom->periodic[k] ? 1 : 0;
        gg->lo[k] = dom->lo[k];
        gg->hi[k] = dom->hi[k];
        volatile float L = dom->hi[k] - dom->lo[k];
        if (!(L > 0.f) || !isfinite(L)) return SPH_E_DOMAIN;
        gg->L[k] = L;
        gg->L_d[k] = (double)L;
        gg->lo_d[k] = (double)dom->lo[k];
        double ratio = (double)L / (double)dom->cell_size;
        int limit = dom->dim == 3 ? 1023 : 65535;
        if (gg->periodic[k]) {
            double f = floor(ratio);
            if (f < 3.0) return SPH_E_DOMAIN;
            if (f > limit) return SPH_E_DOMAIN;
            gg->ncell[k] = (int)f;
            gg->edge[k] = (double)L / f;
        } else {
            double c = ceil(ratio);
            if (c < 1.0) c = 1.0;
            if (c > limit) return SPH_E_DOMAIN;
            gg->ncell[k] = (int)c;
            gg->edge[k] = (double)dom->cell_size;
        }
        if (gg->ncell[k] > maxnc) maxnc = gg->ncell[k];
        tot *= gg->ncell[k];
    }
    if (tot > ((int64_t)1 << 28)) return SPH_E_DOMAIN;
    gg->bits = ceil_log2(maxnc);
    if (gg->bits < 1) gg->bits = 1;
    *ncells_total = tot;
    return SPH_OK;
}

extern "C" int sph_build_cells(sph_ctx *ctx, const sph_domain *dom, const float *x, const float *h, int64_t n,
                               sph_stream_t stream)
{
    if (!ctx || !dom || !x || !h || n <= 0 || n >= ((int64_t)1 << 31)) return SPH_E_INVALID;
    ctx->cells_ready = false;
    ctx->lists_ready = false;
    ctx->rk_lists_prepared = false;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    GridGeom gg;
    int64_t ncells;
    SPH_TRY(make_geom(dom, &gg, &ncells));
    ctx->geom = gg;
    ctx->dom_last = *dom;
    ctx->ncells_total = ncells;
    ctx->n = n;
    ctx->last_stream = st;

    const int64_t nchunks = (n + kChunk - 1) / kChunk;
    SPH_TRY(ctx->key_a.reserve((size_t)n * 4));
    SPH_TRY(ctx->key_b.reserve((size_t)n * 4));
    SPH_TRY(ctx->idx_a.reserve((size_t)n * 4));
    SPH_TRY(ctx->idx_b.reserve((size_t)n * 4));
    SPH_TRY(ctx->hist.reserve((size_t)nchunks * kRsMaxBins * 4));
    SPH_TRY(ctx->perm.reserve((size_t)n * 4));
    SPH_TRY(ctx->inv_perm.reserve((size_t)n * 4));
    SPH_TRY(ctx->pos_s.reserve((size_t)n * 16));
    SPH_TRY(ctx->cell_start.reserve((size_t)ncells * 4));
    SPH_TRY(ctx->cell_end.reserve((size_t)ncells * 4));
    SPH_TRY(ctx->stats.reserve(64));

    const uint32_t init_stats[4] = {0u, 0u, 0x7f7fffffu, 0u};
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->stats.p, init_stats, sizeof(init_stats), cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemsetAsync(ctx->cell_start.p, 0, (size_t)ncells * 4, st));
    SPH_CUDA_TRY(cudaMemsetAsync(ctx->cell_end.p, 0, (size_t)ncells * 4, st));

    const unsigned nblk = (unsigned)((n + kThreads - 1) / kThreads);
    {
        KScope ks(ctx, SPH_K_KEY, 1, st);
        k_wrap_key<<<nblk, kThreads, 0, st>>>(x, h, n, gg, ctx->key_a.as<uint32_t>(), ctx->stats.as<uint32_t>());
    }

    // LSD radix passes over the used key bits
    const int keybits = gg.bits * gg.dim;
    const int passes = (keybits + kRsMaxBits - 1) / kRsMaxBits;
    const int dbits = (keybits + passes - 1) / passes;           // <= kRsMaxBits
    uint32_t *kin = ctx->key_a.as<uint32_t>(), *kout = ctx->key_b.as<uint32_t>();
    uint32_t *vin = nullptr, *vout = ctx->idx_b.as<uint32_t>();
    uint32_t *vother = ctx->idx_a.as<uint32_t>();
    const unsigned rblk = (unsigned)((nchunks + kRsWarps - 1) / kRsWarps);
    for (int p = 0; p < passes; ++p) {
        KScope ks(ctx, SPH_K_SORT, 5, st);
        k_radix_hist<<<rblk, kRsWarps * 32, 0, st>>>(kin, n, dbits * p, dbits, nchunks, ctx->hist.as<uint32_t>());
        SPH_TRY(sph_scan_u32(ctx, ctx->hist.as<uint32_t>(), ctx->hist.p, false, nchunks << dbits, st));
        k_radix_scatter<<<rblk, kRsWarps * 32, 0, st>>>(kin, vin, kout, vout, n, dbits * p, dbits, nchunks, ctx->hist.as<uint32_t>());
        uint32_t *t = kin;
        kin = kout;
        kout = t;
        uint32_t *nv = vin ? vin : vother;
        vin = vout;
        vout = nv;
    }
    // kin / vin now hold the sorted keys and the sorted caller indices
    SPH_TRY(ctx->key_sorted.reserve((size_t)n * 4));
    {
        KScope ks(ctx, SPH_K_REORDER, 1, st);
        SPH_CUDA_TRY(cudaMemcpyAsync(ctx->key_sorted.p, kin, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
        k_reorder<<<nblk, kThreads, 0, st>>>(x, h, n, gg, ctx->key_sorted.as<uint32_t>(), vin, ctx->perm.as<uint32_t>(),
                                             ctx->inv_perm.as<uint32_t>(), ctx->pos_s.as<float4>(),
                                             ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>());
    }
    SPH_CUDA_TRY(cudaGetLastError());
    ctx->cells_ready = true;
    return SPH_OK;
}

// x: current positions; h: NULL, or the current support radii (lists built for other radii are reported invalid)
int sph_lists_valid_impl(sph_ctx *ctx, const float *x, const float *h, float skin_needed, int32_t *valid_out,
                         float *max_disp_out, cudaStream_t st)
{
    const int64_t n = ctx->n;
    uint32_t *slot = ctx->stats.as<uint32_t>() + 12;
    SPH_CUDA_TRY(cudaMemsetAsync(slot, 0, 4, st));
    {
        KScope ks(ctx, SPH_K_KEY, 1, st);
        k_max_displacement<<<(unsigned)((n + kThreads - 1) / kThreads), kThreads, 0, st>>>(
            x, h, n, ctx->geom, ctx->inv_perm.as<uint32_t>(), ctx->pos_s.as<float4>(), slot);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    uint32_t *hp = reinterpret_cast<uint32_t *>(ctx->h_pinned + 14);
    SPH_CUDA_TRY(cudaMemcpyAsync(hp, slot, 4, cudaMemcpyDeviceToHost, st));
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    float D;
    memcpy(&D, hp, 4);
    if (max_disp_out) *max_disp_out = D;
    if (valid_out) {
        const double width = ((double)ctx->search_scale - 1.0 - (double)skin_needed) * (double)ctx->hmin;
        *valid_out = (2.0 * (double)D <= width) ? 1 : 0;
    }
    return SPH_OK;
}

extern "C" int sph_lists_valid(sph_ctx *ctx, const float *x, float skin_needed, int32_t *valid_out, float *max_disp_out,
                               sph_stream_t stream)
{
    if (!ctx || !x || !(skin_needed >= 0.f)) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    return sph_lists_valid_impl(ctx, x, nullptr, skin_needed, valid_out, max_disp_out, st);
}

// ------------------------------------------------------------------------------------------ allocation-free prefix sum
// Step N6 (exclusive scan of the per-row counts -> 64-bit CSR offsets, App. B step 2) for callers that
// must not allocate: CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same three kernels as
// sph_scan_u32 above; the block sums, which that path keeps in a context buffer that grows on demand, live here in a
// file-scope device array of fixed size (16384 x 8 B = 128 KiB, held by every GPU that loads the library until exit).
//
// In host code `g_scan_noalloc` is the host-side stand-in of the symbol, NOT a device address: the address the kernels
// get is looked up once per device, with that device current, by cudaGetSymbolAddress.
constexpr int64_t kNoAllocMaxCount = (int64_t)SPH_PREFIX_SUM_NOALLOC_MAX;
constexpr int64_t kNoAllocMaxBlocks = (kNoAllocMaxCount + kScanTile - 1) / kScanTile;
static __device__ __align__(256) unsigned long long g_scan_noalloc[kNoAllocMaxBlocks];

namespace {
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
unsigned long long *g_noalloc_ptr[kNoAllocMaxDevices] = {};
}

extern "C" int sph_prefix_sum_noalloc(int device, const uint32_t *counts, int64_t *offsets, int64_t n, sph_stream_t stream)
{
    if (device < 0 || device >= kNoAllocMaxDevices || n < 0) return SPH_E_INVALID;
    if (n > kNoAllocMaxCount) return SPH_E_TOO_LARGE;
    if (n > 0 && (!counts || !offsets)) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(device));
    unsigned long long *sums = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_ptr[device]) {
            void *p = nullptr;
            SPH_CUDA_TRY(cudaGetSymbolAddress(&p, g_scan_noalloc));     // this device's copy of the array
            if (!p) return SPH_E_CUDA;
            g_noalloc_ptr[device] = static_cast<unsigned long long *>(p);
        }
        sums = g_noalloc_ptr[device];
    }
    if (n == 0) return SPH_OK;                                          // set-up only
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t nb = (n + kScanTile - 1) / kScanTile;
    // every entry of sums[0, nb) is overwritten by k_scan_reduce before it is read and nothing beyond nb is read, so
    // the contents a previous call left behind need no clearing
    k_scan_reduce<<<(unsigned)nb, kScanThreads, 0, st>>>(counts, n, sums);
    k_scan_sums<<<1, kScanThreads, 0, st>>>(sums, nb);
    k_scan_apply<long long><<<(unsigned)nb, kScanThreads, 0, st>>>(counts, reinterpret_cast<long long *>(offsets), n, sums, 1);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}
