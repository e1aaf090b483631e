// sph_pairs_tile.cu -- the pair-sum kernels D, R1, B1 (+ B2 stage 1) of SURVEY.md 8(a) on the cell-block
// decomposition of sph_tiles.cuh.  One CTA per tile:
//   1. the sorted state of the tile's halo ((B+2)^d cells, each a contiguous run of the sorted SoA) is staged in
//      shared memory, positions shifted by -+L across periodic seams (no minimum image in the inner loop);
//   2. GS lanes share a row.  The uint16 halo indices of the rows a warp works on next (2 B per pair, the only
//      per-pair HBM traffic) are prefetched one pass ahead into a per-warp shared-memory ring with cp.async, so the
//      inner loop contains no global load: LDS.U16 index -> LDS.128 gathers of the neighbour state
//      (~10 shared-memory wavefronts per 32 pairs instead of ~32 L1 wavefronts of global gathers, profiles/r01_b);
//   3. shuffle reduction inside the lane group, one writer per row.  No float atomics; fixed summation order.
// Formulas: include/sph.h header comment and DESIGN.md section 2 (Eq.8, 9, 12, 40, 42, 7).
#include "sph_internal.cuh"
#include "sph_tiles.cuh"
#include "sph_pair_math.cuh"

#include <math.h>

namespace {

constexpr int kPtMaxWarps = 16;      // launch bound of the light pair kernels (<= 128 registers)
constexpr int kVjpMaxWarps = 21;     // k_vjp_tile: the bound of 672 threads caps it at 96 registers, so that 20 warps fit one SM

template <int GS>
__device__ __forceinline__ float group_sum(float v)
{
#pragma unroll
    for (int o = GS / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sums four per-lane values over the GS lanes of a group with 2 + 1 + log2(GS/4) shuffles instead of 4 log2(GS): the
// first two butterfly steps halve the number of values a lane carries.  Lane gl ends up with the total of component
// q = 2 [gl & GS/2] + [gl & GS/4]; the lanes with (gl & (GS/4 - 1)) == 0 are the four writers.  Fixed order: deterministic.
template <int GS>
__device__ __forceinline__ float group_sum4(float v0, float v1, float v2, float v3, int gl)
{
    static_assert(GS >= 4, "four components need four lanes");
    const bool hi = (gl & (GS / 2)) != 0, mid = (gl & (GS / 4)) != 0;
    float a = (hi ? v2 : v0) + __shfl_xor_sync(0xffffffffu, hi ? v0 : v2, GS / 2);
    float b = (hi ? v3 : v1) + __shfl_xor_sync(0xffffffffu, hi ? v1 : v3, GS / 2);
    float c = (mid ? b : a) + __shfl_xor_sync(0xffffffffu, mid ? a : b, GS / 4);
#pragma unroll
    for (int o = GS / 8; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    return c;
}

// ------------------------------------------------------------------------------------------ staging
__device__ __forceinline__ void cp_async16(uint32_t smem_addr, const void *gptr)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async8(uint32_t smem_addr, const void *gptr)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t smem_addr, const void *gptr)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Bulk-copy staging (SPH_OPT_STAGE_BULK, include/sph.h): one cp.async.bulk per halo cell and float4 array instead of one
// 16-byte cp.async per particle, all completing on one mbarrier of the CTA (a tile is staged once, so phase 0 only).
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "SPH_MBAR_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@p bra SPH_MBAR_DONE;\n"
                 "bra SPH_MBAR_WAIT;\n"
                 "SPH_MBAR_DONE:\n"
                 "}\n" ::"r"(smem_u32(bar)), "r"(parity)
                 : "memory");
}

// Copies the halo of the tile (every halo cell is one contiguous run of the sorted arrays) into shared memory with
// cp.async: no registers, every copy of the CTA in flight at once.  Null sources are skipped (compile time).
__device__ __forceinline__ void stage_halo(const TileTab &tt, const float4 *__restrict__ g0, float4 *d0,
                                           const float4 *__restrict__ g1, float4 *d1, const float4 *__restrict__ g2,
                                           float4 *d2, const float2 *__restrict__ gc, float2 *dc,
                                           const float *__restrict__ gf, float *df, uint64_t *bar = nullptr,
                                           int hc_lo = 0, int hc_hi = -1, uint32_t q_lo = 0)
{
    // [hc_lo, hc_hi): the halo cells to stage (default: all); the particle with halo-linear index q lands at slot q - q_lo
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    if (hc_hi < 0) hc_hi = tt.nh;
    const uint32_t a0 = smem_u32(d0) - q_lo * 16u, a1 = smem_u32(d1) - q_lo * 16u, a2 = smem_u32(d2) - q_lo * 16u,
                   ac = smem_u32(dc) - q_lo * 8u, af = smem_u32(df) - q_lo * 4u;
    if (bar) {
        // the float4 arrays by bulk copies (runs are 16-byte aligned multiples of 16 bytes by construction); the caller has
        // initialised the barrier (count 1) and synchronised.  The float2 / float arrays below stay per-particle copies.
        if (threadIdx.x == 0) mbar_expect_tx(bar, (uint32_t)tt.M * 16u * ((g0 ? 1u : 0u) + (g1 ? 1u : 0u) + (g2 ? 1u : 0u)));
        for (int hc = threadIdx.x; hc < tt.nh; hc += blockDim.x) {
            const uint32_t o0 = tt.h_off[hc], cnt = tt.h_off[hc + 1] - o0, gs = tt.h_start[hc];
            if (cnt == 0) continue;
            if (g0) bulk_g2s(a0 + o0 * 16, g0 + gs, cnt * 16, bar);
            if (g1) bulk_g2s(a1 + o0 * 16, g1 + gs, cnt * 16, bar);
            if (g2) bulk_g2s(a2 + o0 * 16, g2 + gs, cnt * 16, bar);
        }
        g0 = nullptr; g1 = nullptr; g2 = nullptr;
        if (!gc && !gf) return;
    }
    for (int hc = hc_lo + warp; hc < hc_hi; hc += nwarps) {
        const uint32_t o0 = tt.h_off[hc], cnt = tt.h_off[hc + 1] - o0, gs = tt.h_start[hc];
        auto copy = [&](uint32_t q, size_t g) {
            if (g0) cp_async16(a0 + q * 16, g0 + g);
            if (g1) cp_async16(a1 + q * 16, g1 + g);
            if (g2) cp_async16(a2 + q * 16, g2 + g);
            if (gc) cp_async8(ac + q * 8, gc + g);
            if (gf) cp_async4(af + q * 4, gf + g);
        };
        // a cell rarely holds more than 64 particles: two rounds at fixed offsets from one set of addresses, then the rest
        const uint32_t q = o0 + lane;
        const size_t g = (size_t)gs + lane;
        if ((uint32_t)lane < cnt) copy(q, g);
        if ((uint32_t)lane + 32u < cnt) copy(q + 32u, g + 32);
        for (uint32_t l = lane + 64; l < cnt; l += 32) copy(o0 + l, (size_t)gs + l);
    }
    cp_async_commit();
}
// after the copies have landed (wait + __syncthreads): add the periodic shift to the positions of the halo cells
// that lie across a face.  Contains a __syncthreads on seam tiles (uniform per CTA).
template <int DIM>
__device__ __forceinline__ void stage_shift(const TileTab &tt, float4 *d0, int hc_lo = 0, int hc_hi = -1, uint32_t q_lo = 0)
{
    if (!tt.seam) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    if (hc_hi < 0) hc_hi = tt.nh;
    d0 -= q_lo;
    for (int hc = hc_lo + warp; hc < hc_hi; hc += nwarps) {
        const float sx = tt.h_shift[0][hc], sy = tt.h_shift[1][hc], sz = DIM == 3 ? tt.h_shift[2][hc] : 0.f;
        if (sx == 0.f && sy == 0.f && sz == 0.f) continue;
        const uint32_t o0 = tt.h_off[hc], cnt = tt.h_off[hc + 1] - o0;
        for (uint32_t l = lane; l < cnt; l += 32) {
            float4 v = d0[o0 + l];
            v.x += sx;
            v.y += sy;
            if (DIM == 3) v.z += sz;
            d0[o0 + l] = v;
        }
    }
    __syncthreads();
}
// tile-relative row offsets rp[r] = row_ptr[row0 + r] - row_ptr[row0], r = 0..T, and the halo index of every row
__device__ __forceinline__ void stage_rows(const TileTab &tt, const long long *__restrict__ row_ptr, uint32_t *rp,
                                           uint16_t *selfq)
{
    const long long base = row_ptr[tt.row0];
    for (uint32_t r = threadIdx.x; r <= tt.T; r += blockDim.x) rp[r] = (uint32_t)(row_ptr[tt.row0 + r] - base);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    for (int tc = warp; tc < tt.nt; tc += nwarps) {
        const int hc = tt.t_cell[tc];
        const uint32_t o0 = tt.h_off[hc], cnt = tt.h_off[hc + 1] - o0;
        const uint32_t rbase = tt.h_start[hc] - tt.row0;
        for (uint32_t l = lane; l < cnt; l += 32) selfq[rbase + l] = (uint16_t)(o0 + l);
    }
}

// sizes of the shared-memory carve-up of one launch (SmemMap below) and its launch-wide switches
struct TileSizes {
    int mcap, tcap, rb;
    int split;           // k_vjp_tile: 2 = each CTA takes half a tile (one z-layer of a 2x2x2 block), 1 = a whole tile
    int bulk;            // SPH_OPT_STAGE_BULK: k_rhs_tile / k_vjp_tile stage their float4 arrays with cp.async.bulk
};

// ts.split == 2 (3D, 2x2x2-cell tiles): two CTAs per tile, each with the rows of one z-layer of target cells and the three
// z-layers of halo cells around it -- a contiguous range of halo cells, of halo-linear indices and (the sort key is the
// Morton code, z its top bit inside a block) of rows.  A halo particle q is staged at slot q - q_lo, and the gathers use
// base pointers moved back by q_lo, so the list entries are used as they are.  Two resident CTAs instead of one (or three
// instead of two) let one stage its halo while the others compute.
struct TilePart {
    uint32_t row_lo, row_hi, q_lo, q_hi;
    int hc_lo, hc_hi;
};
template <int DIM>
__device__ __forceinline__ int tile_of_block(const TileSizes &ts)
{
    return (DIM == 3 && ts.split == 2) ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
}
template <int DIM>
__device__ __forceinline__ TilePart tile_part(const TileTab &tt, const TileSizes &ts)
{
    TilePart tp{0u, tt.T, 0u, tt.M, 0, tt.nh};
    if (DIM == 3 && ts.split == 2) {
        const int half = (int)(blockIdx.x & 1u), per = tt.tn[0] * tt.tn[1];
        if (half >= tt.tn[2]) tp.row_hi = 0;                    // a tile with one layer only: its first CTA has it all
        else if (tt.tn[2] == 2) {
            tp.row_lo = tt.t_off[half * per];
            tp.row_hi = tt.t_off[(half + 1) * per];
            const int zt = tt.tlo[2] + half, slab = tt.ext[0] * tt.ext[1];
            tp.hc_lo = max(zt - 1, 0) * slab;
            tp.hc_hi = (min(zt + 1, tt.ext[2] - 1) + 1) * slab;
            tp.q_lo = tt.h_off[tp.hc_lo];
            tp.q_hi = tt.h_off[tp.hc_hi];
        }
    }
    SPH_ASSERT(tp.q_hi - tp.q_lo <= (uint32_t)ts.mcap);
    return tp;
}

// ------------------------------------------------------------------------------------------ index ring
// Drives the rows of a tile through `body(r, live, b, e, idx)`: row r of the tile (clamped to T-1; `live` false for
// the padding groups of the last pass), its tile-relative entry range [b,e), and a pointer such that idx[k] is the
// halo index of entry k.  A warp works on RPW = 32/GS consecutive rows per pass; the contiguous index segment of
// its NEXT pass is copied into the other half of its ring (16-byte cp.async chunks) before the current pass is
// processed.  A segment that does not fit the ring is read from global memory directly (correct, slower).
template <int GS, class Body>
__device__ __forceinline__ void tile_row_passes(const TileTab &tt, const uint32_t *rp, uint16_t *ring, int rb,
                                                const uint16_t *__restrict__ col16, long long tilebase, Body body,
                                                uint32_t row_lo = 0, uint32_t row_hi = 0xffffffffu)
{
    // [row_lo, row_hi): the rows of the tile this CTA works on (default: all of them)
    constexpr int RPW = 32 / GS;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int g = lane / GS;
    const uint32_t T = min(tt.T, row_hi);
    const uint32_t step = nwarps * RPW;
    uint16_t *myring = ring + (size_t)warp * 2 * rb;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(myring);

    // 32-bit bookkeeping: entry k of the tile sits at seg[tb7 + k], seg 16-byte aligned (chunks of 8 entries)
    const uint32_t tb7 = (uint32_t)(tilebase & 7ll);
    const uint16_t *seg = col16 + (tilebase - (long long)tb7);
    // copies the segment of the pass that starts at row r0 into half `buf` of the ring; returns its first entry and
    // whether it fitted (the consumer of the pass needs both, one iteration later)
    auto issue = [&](uint32_t r0, int buf, uint32_t &s_out, bool &fits) {
        s_out = 0;
        fits = false;
        if (r0 < T) {
            const uint32_t s = rp[r0], e = rp[min(r0 + RPW, T)];
            const uint32_t c0 = (tb7 + s) >> 3, nchunk = ((tb7 + e + 7u) >> 3) - c0;
            s_out = s;
            fits = nchunk * 8u <= (uint32_t)rb;
            if (fits) {
                const uint16_t *src = seg + (size_t)c0 * 8;
                const uint32_t dst = ring_s + (uint32_t)(buf * rb) * 2u;
                // a segment is rarely longer than 64 chunks: two copies per lane at fixed offsets from one address pair
                const uint16_t *src_l = src + (size_t)lane * 8;
                const uint32_t dst_l = dst + (uint32_t)lane * 16u;
                if ((uint32_t)lane < nchunk) cp_async16(dst_l, src_l);
                if ((uint32_t)lane + 32u < nchunk) cp_async16(dst_l + 512u, src_l + 256);
                for (uint32_t c = lane + 64; c < nchunk; c += 32) cp_async16(dst + c * 16u, src + c * 8u);
            }
        }
        cp_async_commit();
    };
    int buf = 0;
    uint32_t s_cur, s_nxt;
    bool f_cur, f_nxt;
    issue(row_lo + warp * RPW, 0, s_cur, f_cur);
    for (uint32_t r0 = row_lo + warp * RPW; r0 < T; r0 += step, buf ^= 1) {
        issue(r0 + step, buf ^ 1, s_nxt, f_nxt);
        cp_async_wait<1>();
        __syncwarp();
        const uint32_t r = min(r0 + g, T - 1);
        const bool live = r0 + g < T;
        const uint32_t b = rp[r], e = rp[r + 1];
        SPH_ASSERT(r < T && e >= b);
        if (f_cur)
            body(r, live, b, e, (const uint16_t *)(myring + buf * rb + ((tb7 + s_cur) & 7u)) - s_cur);
        else
            body(r, live, b, e, col16 + tilebase);
        __syncwarp();
        s_cur = s_nxt;
        f_cur = f_nxt;
    }
    cp_async_wait<0>();
}

// shared-memory load of a particle record (layout: sph_pair_math.cuh)
// UM (3D, uniform mass m0 and uniform h): s2 is not staged at all -- V = m0/rho costs one MUFU and one multiply against
// a third gather with its bank conflicts (the shared-memory data pipe is the binding unit, profiles/r01_g)
template <int DIM, bool UM = false>
__device__ __forceinline__ Part load_part(const float4 *s0, const float4 *s1, const float2 *s2, uint32_t j, float m0 = 0.f,
                                          float H = 0.f)
{
    const float4 a = s0[j], b = s1[j];
    if (DIM == 3) {
        if (UM) return part_unpack<3>(a, b, m0 * fast_rcp(a.w), H);
        const float2 c = s2[j];
        return part_unpack<3>(a, b, c.x, c.y);
    }
    return part_unpack<DIM>(a, b);
}

// shared-memory carve-up: A, B (float4[mcap]), [cot float4[mcap]], C (float2[mcap], 3D only), rp[tcap+1],
// selfq[tcap], index ring [nwarps][2][rb]
template <int DIM>
struct SmemMap {
    float4 *A, *B, *cot;
    float2 *C;
    uint32_t *rp;
    uint16_t *selfq, *ring;
    // b_bytes: bytes per halo particle of the B slot (16; 4 when a kernel keeps one float there, as the density does)
    __device__ SmemMap(unsigned char *base, const TileSizes &ts, bool with_cot, bool with_C = true, int b_bytes = 16)
    {
        size_t o = 0;
        A = reinterpret_cast<float4 *>(base + o); o += (size_t)ts.mcap * 16;
        B = reinterpret_cast<float4 *>(base + o); o += (size_t)ts.mcap * b_bytes;
        cot = reinterpret_cast<float4 *>(base + o); if (with_cot) o += (size_t)ts.mcap * 16;
        C = reinterpret_cast<float2 *>(base + o); if (DIM == 3 && with_C) o += (size_t)ts.mcap * 8;
        rp = reinterpret_cast<uint32_t *>(base + o); o += (size_t)(ts.tcap + 4) * 4;
        selfq = reinterpret_cast<uint16_t *>(base + o); o += (size_t)ts.tcap * 2;
        o = (o + 15) & ~(size_t)15;
        ring = reinterpret_cast<uint16_t *>(base + o);
    }
};

// ------------------------------------------------------------------------------------------ D: density
// smem: A = {x,y,z,h}[mcap], Ms = m[mcap] (in the B slot), rp, selfq, ring
// UM: all masses equal (device flag `um`, written by sph_density's own gather kernel: the launch whose turn it is not
// returns at once, as in k_rhs_tile): the masses are neither staged nor gathered, rho_i = m_0 sum_j W_ij with m_0 = m[0]
template <int DIM, int GS, bool VARH, bool UM>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_density_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ pos_s, const float *__restrict__ m_s,
               const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
               const long long *__restrict__ row_ptr, const uint16_t *__restrict__ col16,
               const uint32_t *__restrict__ perm, float *__restrict__ rho_out, const uint32_t *__restrict__ um,
               const float *__restrict__ m_caller)
{
    if (um && (um[0] != 0u) != UM) return;
    const float m0 = UM ? __ldg(m_caller) : 0.f;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SmemMap<DIM> sm(smem_raw, ts, false, false, UM ? 0 : 4);     // 20 (16) bytes per halo particle: three CTAs per SM at C3
    float *Ms = reinterpret_cast<float *>(sm.B);
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    stage_halo(tt, pos_s, sm.A, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, UM ? nullptr : m_s, Ms);
    stage_rows(tt, row_ptr, sm.rp, sm.selfq);
    cp_async_wait<0>();
    __syncthreads();
    stage_shift<DIM>(tt, sm.A);
    const int gl = (threadIdx.x & 31) % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const float4 *A = sm.A;
    const uint16_t *selfq = sm.selfq;
    const uint32_t row0 = tt.row0;
    tile_row_passes<GS>(tt, sm.rp, sm.ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e, const uint16_t *idx) {
            const float4 pi = A[selfq[r]];
            float acc = 0.f;
#pragma unroll 4
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const float4 pj = A[j];
                const float d0 = pi.x - pj.x, d1 = pi.y - pj.y, d2 = DIM == 3 ? pi.z - pj.z : 0.f;
                const float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
                const float q = fast_sqrt(r2) * hc.invH;
                const float t = fmaxf(1.0f - q, 0.f);
                const float t2 = t * t, t6 = t2 * t2 * t2;
                const float w = hc.cW * t6 * fmaf(q, fmaf(q, 35.0f / 3.0f, 6.0f), 1.0f);   // Eq.25/27
                acc = UM ? acc + w : fmaf(Ms[j], w, acc);
            }
            acc = group_sum<GS>(acc);
            if (gl == 0 && live) rho_out[perm[row0 + r]] = UM ? m0 * acc : acc;
        });
}

// ------------------------------------------------------------------------------------------ D^T: density adjoint
// x_bar_i = sum_j (rb_i m_j + rb_j m_i) G_ij d_ij,  m_bar_i = sum_j rb_j W_ij   (include/sph.h sph_density_vjp;
// PAPER.md:242, 353 Eq.21).  smem: A = {x,y,z,h}[mcap], MR = {m, rho_bar}[mcap] (in the B slot), rp, selfq, ring
template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_density_vjp_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ pos_s, const float2 *__restrict__ mr_s,
                   const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
                   const long long *__restrict__ row_ptr, const uint16_t *__restrict__ col16,
                   const uint32_t *__restrict__ perm, float *__restrict__ xb_out, float *__restrict__ mb_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SmemMap<DIM> sm(smem_raw, ts, false);
    float2 *MR = reinterpret_cast<float2 *>(sm.B);
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    stage_halo(tt, pos_s, sm.A, nullptr, nullptr, nullptr, nullptr, mr_s, MR, nullptr, nullptr);
    stage_rows(tt, row_ptr, sm.rp, sm.selfq);
    cp_async_wait<0>();
    __syncthreads();
    stage_shift<DIM>(tt, sm.A);
    const int gl = (threadIdx.x & 31) % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const float4 *A = sm.A;
    const uint16_t *selfq = sm.selfq;
    const uint32_t row0 = tt.row0;
    tile_row_passes<GS>(tt, sm.rp, sm.ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e, const uint16_t *idx) {
            const uint32_t qi = selfq[r];
            const float4 pi = A[qi];
            const float2 ai = MR[qi];                          // {m_i, rho_bar_i}
            float x0 = 0.f, x1 = 0.f, x2 = 0.f, mb = 0.f;
#pragma unroll 2
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const float4 pj = A[j];
                const float2 aj = MR[j];
                const float d0 = pi.x - pj.x, d1 = pi.y - pj.y, d2 = DIM == 3 ? pi.z - pj.z : 0.f;
                const float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
                const float q = fast_sqrt(r2) * hc.invH;
                const float t = fmaxf(1.0f - q, 0.f);
                const float t2 = t * t, t4 = t2 * t2;
                const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                             // Eq.29
                const float w = hc.cW * (t4 * t2) * fmaf(q, fmaf(q, 35.0f / 3.0f, 6.0f), 1.0f);     // Eq.25/27
                const float c = fmaf(ai.y, aj.x, aj.y * ai.x) * G;
                x0 = fmaf(c, d0, x0);
                x1 = fmaf(c, d1, x1);
                if (DIM == 3) x2 = fmaf(c, d2, x2);
                mb = fmaf(aj.y, w, mb);
            }
            x0 = group_sum<GS>(x0);
            x1 = group_sum<GS>(x1);
            if (DIM == 3) x2 = group_sum<GS>(x2);
            mb = group_sum<GS>(mb);
            if (gl == 0 && live) {
                const int64_t i = perm[row0 + r];
                xb_out[i * DIM] = x0;
                xb_out[i * DIM + 1] = x1;
                if (DIM == 3) xb_out[i * DIM + 2] = x2;
                if (mb_out) mb_out[i] = mb;
            }
        });
}

// ------------------------------------------------------------------------------------------ kernel renormalisation
// moments of PAPER.md:524-528 Eq.44/45: M_i = -sum_j V_j G_ij d d^T (symmetric) and b_i = sum_j V_j (A_j - A_i) G_ij d,
// written as a sorted-order record (3D: 3 float4, 2D: 2 float4; layout in sph_pairs.cu) for k_renorm_solve.
// smem: A = {x,y,z,h}[mcap], VA = {V, A}[mcap] (in the B slot), rp, selfq, ring
template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_renorm_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ pos_s, const float2 *__restrict__ va_s,
              const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
              const long long *__restrict__ row_ptr, const uint16_t *__restrict__ col16, float4 *__restrict__ mom)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SmemMap<DIM> sm(smem_raw, ts, false);
    float2 *VA = reinterpret_cast<float2 *>(sm.B);
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    stage_halo(tt, pos_s, sm.A, nullptr, nullptr, nullptr, nullptr, va_s, VA, nullptr, nullptr);
    stage_rows(tt, row_ptr, sm.rp, sm.selfq);
    cp_async_wait<0>();
    __syncthreads();
    stage_shift<DIM>(tt, sm.A);
    const int gl = (threadIdx.x & 31) % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const float4 *A = sm.A;
    const uint16_t *selfq = sm.selfq;
    const uint32_t row0 = tt.row0;
    tile_row_passes<GS>(tt, sm.rp, sm.ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e, const uint16_t *idx) {
            const uint32_t qi = selfq[r];
            const float4 pi = A[qi];
            const float Ai = VA[qi].y;
            float mxx = 0.f, mxy = 0.f, mxz = 0.f, myy = 0.f, myz = 0.f, mzz = 0.f, b0 = 0.f, b1 = 0.f, b2 = 0.f;
#pragma unroll 2
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const float4 pj = A[j];
                const float2 aj = VA[j];                           // {V_j, A_j}
                const float d0 = pi.x - pj.x, d1 = pi.y - pj.y, d2 = DIM == 3 ? pi.z - pj.z : 0.f;
                const float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
                const float q = fast_sqrt(r2) * hc.invH;
                const float t = fmaxf(1.0f - q, 0.f);
                const float t2 = t * t, t4 = t2 * t2;
                const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                             // Eq.29
                const float c = aj.x * G, dA = aj.y - Ai;
                const float c0 = c * d0, c1 = c * d1, c2 = c * d2;
                mxx = fmaf(-c0, d0, mxx);
                mxy = fmaf(-c0, d1, mxy);
                myy = fmaf(-c1, d1, myy);
                b0 = fmaf(c0, dA, b0);
                b1 = fmaf(c1, dA, b1);
                if (DIM == 3) {
                    mxz = fmaf(-c0, d2, mxz);
                    myz = fmaf(-c1, d2, myz);
                    mzz = fmaf(-c2, d2, mzz);
                    b2 = fmaf(c2, dA, b2);
                }
            }
            mxx = group_sum<GS>(mxx); mxy = group_sum<GS>(mxy); myy = group_sum<GS>(myy);
            b0 = group_sum<GS>(b0); b1 = group_sum<GS>(b1);
            if (DIM == 3) {
                mxz = group_sum<GS>(mxz); myz = group_sum<GS>(myz); mzz = group_sum<GS>(mzz); b2 = group_sum<GS>(b2);
            }
            if (gl == 0 && live) {
                const size_t row = (size_t)row0 + r;
                if (DIM == 3) {
                    mom[row * 3] = make_float4(mxx, mxy, mxz, myy);
                    mom[row * 3 + 1] = make_float4(myz, mzz, b0, b1);
                    mom[row * 3 + 2] = make_float4(b2, 0.f, 0.f, 0.f);
                } else {
                    mom[row * 2] = make_float4(mxx, mxy, myy, b0);
                    mom[row * 2 + 1] = make_float4(b1, 0.f, 0.f, 0.f);
                }
            }
        });
}

// pair pass of the adjoint of the renormalised gradient (formulas: sph_pairs.cu k_renorm_vjp, sph_pair_math.cuh).
// smem (own carve-up, 60 B per halo particle in 3D, 44 B in 2D): A = {x,y,z,h}, RB = {V, A, b_bar0, b_bar1},
// RC = {b_bar2, Nxx, Nxy, Nxz} (3D only), RD = float2, RE = float; then rp, selfq, ring as in SmemMap
template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_renorm_vjp_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ pos_s, const float4 *__restrict__ rb,
                  const float4 *__restrict__ rc, const float2 *__restrict__ rd, const float *__restrict__ re,
                  const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
                  const long long *__restrict__ row_ptr, const uint16_t *__restrict__ col16,
                  const uint32_t *__restrict__ perm, float *__restrict__ xb_out, float *__restrict__ vb_out,
                  float *__restrict__ ab_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    size_t o = 0;
    float4 *A = reinterpret_cast<float4 *>(smem_raw + o); o += (size_t)ts.mcap * 16;
    float4 *RB = reinterpret_cast<float4 *>(smem_raw + o); o += (size_t)ts.mcap * 16;
    float4 *RC = reinterpret_cast<float4 *>(smem_raw + o); if (DIM == 3) o += (size_t)ts.mcap * 16;
    float2 *RD = reinterpret_cast<float2 *>(smem_raw + o); o += (size_t)ts.mcap * 8;
    float *RE = reinterpret_cast<float *>(smem_raw + o); o += (size_t)ts.mcap * 4;
    uint32_t *rp = reinterpret_cast<uint32_t *>(smem_raw + o); o += (size_t)(ts.tcap + 4) * 4;
    uint16_t *selfq = reinterpret_cast<uint16_t *>(smem_raw + o); o += (size_t)ts.tcap * 2;
    o = (o + 15) & ~(size_t)15;
    uint16_t *ring = reinterpret_cast<uint16_t *>(smem_raw + o);
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    stage_halo(tt, pos_s, A, rb, RB, DIM == 3 ? rc : nullptr, RC, rd, RD, re, RE);
    stage_rows(tt, row_ptr, rp, selfq);
    cp_async_wait<0>();
    __syncthreads();
    stage_shift<DIM>(tt, A);
    const int gl = (threadIdx.x & 31) % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const uint32_t row0 = tt.row0;
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    tile_row_passes<GS>(tt, rp, ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e, const uint16_t *idx) {
            const uint32_t qi = selfq[r];
            const float4 pi = A[qi];
            const RenormRec ri = renorm_rec<DIM>(RB[qi], DIM == 3 ? RC[qi] : zero4, RD[qi], RE[qi]);
            float xb[3] = {0.f, 0.f, 0.f}, vb = 0.f, ab = 0.f;
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const float4 pj = A[j];
                const RenormRec rj = renorm_rec<DIM>(RB[j], DIM == 3 ? RC[j] : zero4, RD[j], RE[j]);
                const float d[3] = {pi.x - pj.x, pi.y - pj.y, DIM == 3 ? pi.z - pj.z : 0.f};
                const float r2 = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
                const float q = fast_sqrt(r2) * hc.invH;
                const float t = fmaxf(1.0f - q, 0.f);
                const float t2 = t * t, t4 = t2 * t2;
                const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                             // Eq.29
                const float K = hc.cK * t4;                                                         // Eq.16
                renorm_vjp_pair<DIM>(ri, rj, d, G, K, xb, vb, ab);
            }
#pragma unroll
            for (int k = 0; k < DIM; ++k) xb[k] = group_sum<GS>(xb[k]);
            vb = group_sum<GS>(vb);
            ab = group_sum<GS>(ab);
            if (gl == 0 && live) {
                const int64_t i = perm ? (int64_t)perm[row0 + r] : (int64_t)(row0 + r);   // null perm: sorted order
#pragma unroll
                for (int k = 0; k < DIM; ++k) xb_out[i * DIM + k] = xb[k];
                if (vb_out) vb_out[i] = vb;
                if (ab_out) ab_out[i] = ab;
            }
        });
}

// ------------------------------------------------------------------------------------------ kernel-gradient sum
// g_i = sum_j a_j G_ij d_ij (VJP = false; smem A = positions, W = a[mcap] in the B slot) and its adjoint (VJP = true;
// smem A, GA = {g_bar, a}[mcap] in the B slot): include/sph.h sph_grad_sum / sph_grad_sum_vjp; Eq.24
template <int DIM, int GS, bool VARH, bool VJP>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_grad_sum_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ pos_s, const float *__restrict__ a_s,
                const float4 *__restrict__ ga_s, const uint32_t *__restrict__ cell_start,
                const uint32_t *__restrict__ cell_end, const long long *__restrict__ row_ptr,
                const uint16_t *__restrict__ col16, const uint32_t *__restrict__ perm, float *__restrict__ v_out,
                float *__restrict__ a_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SmemMap<DIM> sm(smem_raw, ts, false);
    float *Ws = reinterpret_cast<float *>(sm.B);
    const float4 *GA = sm.B;
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    if (VJP) stage_halo(tt, pos_s, sm.A, ga_s, sm.B, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);
    else stage_halo(tt, pos_s, sm.A, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, a_s, Ws);
    stage_rows(tt, row_ptr, sm.rp, sm.selfq);
    cp_async_wait<0>();
    __syncthreads();
    stage_shift<DIM>(tt, sm.A);
    const int gl = (threadIdx.x & 31) % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const float4 *A = sm.A;
    const uint16_t *selfq = sm.selfq;
    const uint32_t row0 = tt.row0;
    tile_row_passes<GS>(tt, sm.rp, sm.ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e, const uint16_t *idx) {
            const uint32_t qi = selfq[r];
            const float4 pi = A[qi];
            float4 gi = make_float4(0.f, 0.f, 0.f, 0.f);
            if (VJP) gi = GA[qi];
            float x0 = 0.f, x1 = 0.f, x2 = 0.f, ab = 0.f;
#pragma unroll 2
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const float4 pj = A[j];
                const float d0 = pi.x - pj.x, d1 = pi.y - pj.y, d2 = DIM == 3 ? pi.z - pj.z : 0.f;
                const float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
                const float q = fast_sqrt(r2) * hc.invH;
                const float t = fmaxf(1.0f - q, 0.f);
                const float t2 = t * t, t4 = t2 * t2;
                const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                             // Eq.29
                if (!VJP) {
                    const float c = Ws[j] * G;
                    x0 = fmaf(c, d0, x0);
                    x1 = fmaf(c, d1, x1);
                    if (DIM == 3) x2 = fmaf(c, d2, x2);
                } else {
                    const float4 gj = GA[j];
                    const float K = hc.cK * t4;                                                     // Eq.16
                    const float dgi = fmaf(d2, gi.z, fmaf(d1, gi.y, d0 * gi.x));
                    const float dgj = fmaf(d2, gj.z, fmaf(d1, gj.y, d0 * gj.x));
                    const float cG = G * gj.w, cGp = G * gi.w;                  // a_j G, a_i G
                    const float cd = K * fmaf(gj.w, dgi, -(gi.w * dgj));        // K (a_j d.gb_i - a_i d.gb_j)
                    x0 += fmaf(cG, gi.x, fmaf(-cGp, gj.x, cd * d0));
                    x1 += fmaf(cG, gi.y, fmaf(-cGp, gj.y, cd * d1));
                    if (DIM == 3) x2 += fmaf(cG, gi.z, fmaf(-cGp, gj.z, cd * d2));
                    ab = fmaf(-G, dgj, ab);
                }
            }
            x0 = group_sum<GS>(x0);
            x1 = group_sum<GS>(x1);
            if (DIM == 3) x2 = group_sum<GS>(x2);
            if (VJP) ab = group_sum<GS>(ab);
            if (gl == 0 && live) {
                const int64_t i = perm[row0 + r];
                v_out[i * DIM] = x0;
                v_out[i * DIM + 1] = x1;
                if (DIM == 3) v_out[i * DIM + 2] = x2;
                if (VJP && a_out) a_out[i] = ab;
            }
        });
}

// ------------------------------------------------------------------------------------------ R1: RHS
// OUT_SORTED: write float4 {a, drho/dt} in sorted order (RK stages); else scatter to the caller's arrays.
// F1: pressure form 1, (p_i + p_j)/(rho_i rho_j), instead of the symmetric Eq.40
// UM: uniform-mass variant (3D, uniform h).  `um` = sph_um_flag: a launch whose UM does not match the flag returns at
// once, so the host can enqueue both variants without knowing the masses (um == nullptr: run unconditionally)
template <int DIM, int GS, bool VARH, bool OUT_SORTED, bool F1, bool UM>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_rhs_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ s0, const float4 *__restrict__ s1,
           const float2 *__restrict__ s2, const uint8_t *__restrict__ kind_s, const uint32_t *__restrict__ cell_start,
           const uint32_t *__restrict__ cell_end, const long long *__restrict__ row_ptr,
           const uint16_t *__restrict__ col16, const uint32_t *__restrict__ perm, float *__restrict__ drho_out,
           float *__restrict__ acc_out, float4 *__restrict__ out4, const uint32_t *__restrict__ um)
{
    static_assert(!UM || (DIM == 3 && !VARH), "the uniform-mass variant is the 3D, uniform-h one");
    if (um && (um[0] != 0u) != UM) return;
    const float m0 = UM ? __uint_as_float(um[1]) : 0.f;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SmemMap<DIM> sm(smem_raw, ts, false, !UM);
    __shared__ TileTab tt;
    // whole tiles: half tiles (k_vjp_tile) were measured for this kernel twice and cost more staging than the third
    // resident CTA hides (profiles/r02_h, r02_i); without them the gathers need no index offset
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    __shared__ uint64_t mbar;
    const bool bulk = ts.bulk != 0;
    if (bulk) {
        if (threadIdx.x == 0) mbar_init(&mbar, 1);
        __syncthreads();
    }
    stage_halo(tt, s0, sm.A, s1, sm.B, nullptr, nullptr, (DIM == 3 && !UM) ? s2 : nullptr, sm.C, nullptr, nullptr,
               bulk ? &mbar : nullptr);
    stage_rows(tt, row_ptr, sm.rp, sm.selfq);
    cp_async_wait<0>();
    if (bulk) mbar_wait(&mbar, 0);
    __syncthreads();
    stage_shift<DIM>(tt, sm.A);
    const int gl = (threadIdx.x & 31) % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const float rho0 = kp.rho0;
    const float umG = m0 * hu.cG, umG5 = umG * 5.0f * hu.invH;      // uniform mass: m0 G = (umG + umG5 r) (1-q)^5
    const float4 *A = sm.A, *B = sm.B;
    const float2 *C = sm.C;
    const uint16_t *selfq = sm.selfq;
    const uint32_t row0 = tt.row0;
    tile_row_passes<GS>(tt, sm.rp, sm.ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e, const uint16_t *idx) {
            const Part pi = load_part<DIM, UM>(A, B, C, selfq[r], m0, kp.H);
            const float ir_i = fast_rcp(pi.rho);
            const float visc_i = rho0 * ir_i;                 // rho0/rho_i of the viscous term
            const float ev_u = hu.eta * visc_i;
            const float Pr_i = pi.P * pi.rho;                 // form 1: p_i/rho_i
            const bool fixed = kind_s[row0 + r] != 0;         // loaded before the pair loop: its latency is hidden
            float sA = 0.f, sD = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll 2
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const Part pj = load_part<DIM, UM>(A, B, C, j, m0, kp.H);
                const float d0 = pi.x[0] - pj.x[0], d1 = pi.x[1] - pj.x[1], d2 = DIM == 3 ? pi.x[2] - pj.x[2] : 0.f;
                const float r2 = fmaf(d2, d2, fmaf(d1, d1, d0 * d0));
                HC hc = hu;
                float ev = ev_u;
                if (VARH) {
                    hc = hc_make<DIM>(fmaxf(pi.h, pj.h), kp);
                    ev = hc.eta * visc_i;
                }
                const float rr = fast_sqrt(r2);
                const float t = fmaxf(fmaf(-hc.invH, rr, 1.0f), 0.f);   // (1-q)+ : skin pairs contribute exactly 0
                const float t2 = t * t, t4 = t2 * t2;
                float s = (pi.v[0] - pj.v[0]) * d0;
                s = fmaf(pi.v[1] - pj.v[1], d1, s);
                if (DIM == 3) s = fmaf(pi.v[2] - pj.v[2], d2, s);
                const float invR = fast_rcp(r2 + hc.e2);
                float cf;
                if (UM && !F1) {
                    // uniform mass, Eq.40: the mass rides on the kernel factor, mG = m0 G, so that V_j G = mG / rho_j and
                    // E G = -mG (P_i + P_j); G alone is never formed (three instructions fewer per pair)
                    const float mG = fmaf(umG5, rr, umG) * (t4 * t);
                    const float VG = mG * fast_rcp(pj.rho);
                    const float q1 = VG * s;
                    sA += q1;
                    sD += VG * (pi.rho - pj.rho) * (r2 * invR);
                    cf = fmaf(ev * invR, q1, -mG * (pi.P + pj.P));
                } else {
                    const float G = hc.cG * fmaf(5.0f * hc.invH, rr, 1.0f) * (t4 * t);
                    const float VG = pj.V * G;
                    // continuity (Eq.9, physical sign) and delta-term (Brookshaw Laplacian of rho)
                    sA = fmaf(VG, s, sA);
                    const float dterm = VG * (pi.rho - pj.rho) * (r2 * invR);
                    sD = VARH ? fmaf(hc.kd, dterm, sD) : sD + dterm;
                    // pressure (Eq.40, symmetric) + viscosity (Eq.7 with the delta-SPH Pi_ij)
                    // E = -m_j e,  e = P_i + P_j (Eq.40)  or  (p_i + p_j)/(rho_i rho_j) = (p_i/rho_i + p_j/rho_i)/rho_j
                    const float mj = UM ? m0 : pj.V * pj.rho;
                    const float E = F1 ? -pj.V * fmaf(pj.P * pj.rho * pj.rho, ir_i, Pr_i) : -mj * (pi.P + pj.P);
                    cf = fmaf(ev * pj.V * s, invR, E) * G;
                }
                a0 = fmaf(cf, d0, a0);
                a1 = fmaf(cf, d1, a1);
                if (DIM == 3) a2 = fmaf(cf, d2, a2);
            }
            const float dr = pi.rho * sA + (VARH ? sD : hu.kd * sD);
            // components {a0, a1, a2, drho} of the row, one per quarter of the lane group
            float val = group_sum4<GS>(a0, a1, a2, dr, gl);
            if ((gl & (GS / 4 - 1)) == 0 && live) {
                const int q = ((gl & (GS / 2)) ? 2 : 0) + ((gl & (GS / 4)) ? 1 : 0);
                const uint32_t row = row0 + r;
                if (q < 3) val = fixed ? 0.f : val + kp.g[q];
                if (OUT_SORTED) {
                    reinterpret_cast<float *>(out4 + row)[q] = val;
                } else {
                    const int64_t i = perm[row];
                    if (q == 3) drho_out[i] = val;
                    else if (q < DIM) acc_out[i * DIM + q] = val;
                }
            }
        });
}

// ------------------------------------------------------------------------------------------ B1: VJP
// Row i evaluates BOTH ordered pairs (i<-j) and (j<-i) of every neighbour j and keeps what lands on i (the list is
// symmetric), so there is no scatter.  The pressure enters through the per-particle P_i = p_i/rho_i^2: its adjoint is
// collected as Z_i and pushed through the EOS once per row.  Per-lane running sums of the scalar-parameter partials
// are reduced per CTA in a fixed order (B2 stage 1); one CTA = one tile = one partials record.
constexpr int kNPartT = 12;   // must match kNPart of sph_pairs.cu (k_reduce_params)

template <int DIM, int GS, bool VARH, bool OUT_SORTED, bool F1, bool UM>
__global__ void __launch_bounds__(kVjpMaxWarps * 32)
k_vjp_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ s0, const float4 *__restrict__ s1,
           const float2 *__restrict__ s2, const float4 *__restrict__ cot, const float4 *__restrict__ eos,
           const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
           const long long *__restrict__ row_ptr, const uint16_t *__restrict__ col16, const uint32_t *__restrict__ perm,
           float *__restrict__ xb_out, float *__restrict__ vb_out, float *__restrict__ rb_out, float4 *__restrict__ xb4,
           float4 *__restrict__ vb4, float *__restrict__ partials, const uint32_t *__restrict__ um)
{
    static_assert(!UM || (DIM == 3 && !VARH), "the uniform-mass variant is the 3D, uniform-h one");
    if (um && (um[0] != 0u) != UM) return;          // see k_rhs_tile
    const float m0 = UM ? __uint_as_float(um[1]) : 0.f;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SmemMap<DIM> sm(smem_raw, ts, true, !UM);
    __shared__ TileTab tt;
    __shared__ float red[kVjpMaxWarps][kNPartT];
    tile_setup<DIM>(tg, tile_of_block<DIM>(ts), cell_start, cell_end, tt);
    const TilePart tp = tile_part<DIM>(tt, ts);
    const uint32_t row_lo = tp.row_lo, row_hi = tp.row_hi, q_lo = tp.q_lo;
    const int hc_lo = tp.hc_lo, hc_hi = tp.hc_hi;
    if (row_hi <= row_lo) {
        if (threadIdx.x < kNPartT) partials[(int64_t)blockIdx.x * kNPartT + threadIdx.x] = 0.f;
        return;
    }
    __shared__ uint64_t mbar;
    const bool bulk = ts.bulk && ts.split != 2;
    if (bulk) {
        if (threadIdx.x == 0) mbar_init(&mbar, 1);
        __syncthreads();
    }
    stage_halo(tt, s0, sm.A, s1, sm.B, cot, sm.cot, (DIM == 3 && !UM) ? s2 : nullptr, sm.C, nullptr, nullptr,
               bulk ? &mbar : nullptr, hc_lo, hc_hi, q_lo);
    stage_rows(tt, row_ptr, sm.rp, sm.selfq);
    cp_async_wait<0>();
    if (bulk) mbar_wait(&mbar, 0);
    __syncthreads();
    stage_shift<DIM>(tt, sm.A, hc_lo, hc_hi, q_lo);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, gl = lane % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const float rho0 = kp.rho0;
    const float4 *A = sm.A - q_lo, *B = sm.B - q_lo, *Ct = sm.cot - q_lo;
    const float2 *C = sm.C - q_lo;
    const uint16_t *selfq = sm.selfq;
    const uint32_t row0 = tt.row0;
    const uint32_t q_hi = tp.q_hi;
    (void)q_hi;
    float S_D1 = 0.f, S_P1 = 0.f, S_PL = 0.f, S_eps = 0.f;                 // per lane, over all its pairs
    float T_E = 0.f, T_0 = 0.f, T_g = 0.f, G0 = 0.f, G1 = 0.f, G2 = 0.f;   // lane 0 of each group, per row
    tile_row_passes<GS>(tt, sm.rp, sm.ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e_in, const uint16_t *idx) {
            const uint32_t qi = selfq[r];
            const Part pi = load_part<DIM, UM>(A, B, C, qi, m0, kp.H);
            const float4 ci = Ct[qi];
            const float lam_i = ci.x, mu_i[3] = {ci.y, ci.z, ci.w};
            const float m_i = UM ? m0 : pi.V * pi.rho, Vi = pi.V, Li = lam_i * pi.rho;
            const uint32_t e = live ? e_in : b;                    // padding groups run no pairs (partials stay clean)
            const float ir_i = 1.0f / pi.rho;
            const float p_i = pi.P * pi.rho * pi.rho;             // form 1: the pressure itself
            float xb[3] = {0.f, 0.f, 0.f}, vb[3] = {0.f, 0.f, 0.f}, rb = 0.f, Z = 0.f, Zr = 0.f;
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j >= q_lo && j < q_hi);
                Part pj = load_part<DIM, UM>(A, B, C, j, m0, kp.H);
                const float4 cj = Ct[j];
                const float lam_j = cj.x, mu_j[3] = {cj.y, cj.z, cj.w};
                const float d[3] = {pi.x[0] - pj.x[0], pi.x[1] - pj.x[1], DIM == 3 ? pi.x[2] - pj.x[2] : 0.f};
                const float r2 = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.h, pj.h), kp);
                const float rr = fast_sqrt(r2);
                const float t = fmaxf(fmaf(-hc.invH, rr, 1.0f), 0.f);
                const float t2 = t * t, t4 = t2 * t2;
                const float G = hc.cG * fmaf(5.0f * hc.invH, rr, 1.0f) * (t4 * t);
                const float K = hc.cK * t4;
                const float w[3] = {pi.v[0] - pj.v[0], pi.v[1] - pj.v[1], DIM == 3 ? pi.v[2] - pj.v[2] : 0.f};
                float s = w[0] * d[0];
                s = fmaf(w[1], d[1], s);
                if (DIM == 3) s = fmaf(w[2], d[2], s);
                const float invR = fast_rcp(r2 + hc.e2);
                const float u = r2 * invR;
                const float ir_j = fast_rcp(pj.rho);
                const float m_j = UM ? m0 : pj.V * pj.rho;
                if (UM) pj.V = m0 * ir_j;                           // the same MUFU result load_part used
                const float drho = pi.rho - pj.rho;
                // pressure pair factor e: E = -m_j e, E' = -m_i e;  e = P_i + P_j (Eq.40) or (p_i + p_j)/(rho_i rho_j)
                const float W2 = ir_i * ir_j;
                const float Psum = F1 ? fmaf(pj.P * pj.rho, pj.rho, p_i) * W2 : pi.P + pj.P;
                float mm = mu_i[0] * d[0];                          // mu_i . d
                mm = fmaf(mu_i[1], d[1], mm);
                if (DIM == 3) mm = fmaf(mu_i[2], d[2], mm);
                float mmj = mu_j[0] * d[0];                         // mu_j . d   (pair (j<-i) uses -d: mmp = -mmj)
                mmj = fmaf(mu_j[1], d[1], mmj);
                if (DIM == 3) mmj = fmaf(mu_j[2], d[2], mmj);
                // The two ordered pairs (i<-j) and (j<-i) of SURVEY.md 8(c-7), with their common factors pulled out
                // (G, eta rho0 G / R, kd drho / R); primes mark the (j<-i) quantities, which use -d, -w and the roles
                // of i and j swapped.
                const float p = pj.V * ir_i, pp = Vi * ir_j;        // V_j/rho_i, V_i/rho_j
                const float ri = rho0 * invR;
                const float t0 = ri * s;
                const float Phi1 = t0 * p, Phi1p = t0 * pp;         // Phi/eta, Phi'/eta
                const float Phi = hc.eta * Phi1, Phip = hc.eta * Phi1p;
                const float zz = fmaf(m_j, mm, -(m_i * mmj));       // m_j mm + m_i mm'      (-dL/dP share of the pair)
                const float q2 = fmaf(mm, Phi, -(mmj * Phip));      // mm Phi + mm' Phi'
                const float Lj = lam_j * pj.rho;
                const float aV = lam_i * pj.V, bV = lam_j * Vi;
                const float q1 = aV - bV;
                const float du = drho * u;
                const float kr = hc.kd * drho * invR;
                const float D = kr * r2;                            // kd drho r2/R        (delta-term / (V G))
                const float Dp = kr * (hc.e2 * invR);               // kd drho e2/R^2      (its r2 derivative)
                const float gG = hc.eta * ri * G;
                const float LL = fmaf(pj.V, Li, Vi * Lj);           // lam_i rho_i V_j + lam_j rho_j V_i
                const float mp = fmaf(mm, p, -(mmj * pp));
                const float cs = fmaf(G, LL, gG * mp);              // sbar + sbar'
                const float X1 = fmaf(Dp, q1, -(invR * q2));        // (r2bar + r2bar') / G
                const float X2 = fmaf(s, LL, fmaf(D, q1, fmaf(-Psum, zz, q2)));   // Gbar + Gbar'
                const float cd = fmaf(G + G, X1, K * X2);
                const float ce = G * fmaf(-m_j, Psum, Phi), cep = G * fmaf(-m_i, Psum, Phip);   // (E+Phi) G, (E'+Phi') G
#pragma unroll
                for (int kk = 0; kk < DIM; ++kk) {
                    xb[kk] = fmaf(cs, w[kk], fmaf(cd, d[kk], fmaf(ce, mu_i[kk], fmaf(-cep, mu_j[kk], xb[kk]))));
                    vb[kk] = fmaf(cs, d[kk], vb[kk]);
                }
                const float kdu = hc.kd * u;
                const float y2 = fmaf(fmaf(pj.rho, s, -D), ir_i, kdu);
                rb = fmaf(G, fmaf(aV, s + kdu, -fmaf(bV, y2, ir_i * q2)), rb);
                if (F1) {
                    const float Gzz = G * zz;
                    Z = fmaf(Gzz, W2, Z);                           // -dL/dp_i
                    Zr = fmaf(Gzz, Psum, Zr);                       // explicit 1/(rho_i rho_j) dependence of e
                } else {
                    Z = fmaf(G, zz, Z);                             // -dL/dP_i
                }
                // ---- scalar parameters, ordered pair (i<-j) only (each ordered pair is owned by one row); the
                // H-dependent factors (2 ell, ell, H^2) are applied after the loops when h is uniform
                const float Gdu = G * du;
                const float xphi1 = mm * G * Phi1;
                const float se = invR * G * fmaf(aV, D, mm * Phi);
                S_P1 += xphi1;
                if (VARH) {
                    S_D1 = fmaf(aV * Gdu, 2.0f * hc.ell, S_D1);
                    S_PL = fmaf(xphi1, hc.ell, S_PL);
                    S_eps = fmaf(se, hc.H2, S_eps);
                } else {
                    S_D1 = fmaf(aV, Gdu, S_D1);
                    S_eps += se;
                }
            }
#pragma unroll
            for (int kk = 0; kk < DIM; ++kk) {
                xb[kk] = group_sum<GS>(xb[kk]);
                vb[kk] = group_sum<GS>(vb[kk]);
            }
            rb = group_sum<GS>(rb);
            Z = group_sum<GS>(Z);
            if (F1) Zr = group_sum<GS>(Zr);
            if (gl == 0 && live) {
                const uint32_t row = row0 + r;
                const float4 ei = eos[row];                          // {dP/drho, dP/drho0, dP/dgamma, m}
                if (F1) {
                    // the EOS enters through p = P rho^2: dp/drho = (dP/drho + 2 P/rho) rho^2, dp/dtheta = dP/dtheta rho^2
                    const float r2i = pi.rho * pi.rho;
                    rb += fmaf(-(ei.x + 2.0f * pi.P * ir_i) * r2i, Z, ir_i * Zr);
                    T_E += p_i * Z;
                    T_0 += ei.y * r2i * Z;
                    T_g += ei.z * r2i * Z;
                } else {
                    rb -= ei.x * Z;                                  // rho_bar_i += Pbar_i dP/drho, Pbar_i = -Z_i
                    T_E += pi.P * Z;
                    T_0 += ei.y * Z;
                    T_g += ei.z * Z;
                }
                G0 += mu_i[0]; G1 += mu_i[1]; G2 += mu_i[2];
                if (OUT_SORTED) {
                    xb4[row] = make_float4(xb[0], xb[1], xb[2], rb);
                    vb4[row] = make_float4(vb[0], vb[1], vb[2], 0.f);
                } else {
                    const int64_t i = perm[row];
#pragma unroll
                    for (int kk = 0; kk < DIM; ++kk) {
                        xb_out[i * DIM + kk] = xb[kk];
                        vb_out[i * DIM + kk] = vb[kk];
                    }
                    rb_out[i] = rb;
                }
            }
        }, row_lo, row_hi);
    // S_D1 = sum lam_i D_ij/(delta c0), S_PL = sum ell xphi1, S_eps = d/d eps: factors left out of the loop
    if (!VARH) {
        S_D1 *= 2.0f * hu.ell;
        S_PL = hu.ell * S_P1;
        S_eps *= -2.0f * kp.eps * hu.H2;
    } else {
        S_eps *= -2.0f * kp.eps;
    }
    // B2 stage 1: fixed-order CTA reduction of the ten partial sums
    float vals[10] = {S_D1, S_P1, S_PL, S_eps, T_E, T_0, T_g, G0, G1, G2};
#pragma unroll
    for (int k = 0; k < 10; ++k) {
        float v = vals[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < kNPartT) {
        float v = 0.f;
        if (threadIdx.x < 10)
            for (int w = 0; w < nwarps; ++w) v += red[w][threadIdx.x];
        partials[(int64_t)blockIdx.x * kNPartT + threadIdx.x] = v;
    }
}

// ------------------------------------------------------------------------------------------ delta-term of [43]
// Second part of the delta-SPH diffusion with the renormalised density gradient (sph_params.delta_form = 1; PAPER.md:103,
// 85, 524-530; reading R17):  X_ij = -delta l_ij c0 V_j (g_i + g_j).d G,  g = <grad rho>^L.
// smem: A = {x,y,z,h} (current positions), B = {g_x,g_y,g_z,V}, ADJ: C = {lambda, rho} (float2).
//   ADJ = false: drho_i += sum_j X_ij                                   (added to the caller's array or to out4[row].w)
//   ADJ = true : gather form of the adjoint for the cotangent lambda (both ordered pairs of every neighbour in the
//                owner's row; w = lambda_i V_j - lambda_j V_i, S = (g_i+g_j).d, Q = (g_i+g_j) G + S K d):
//                x_bar_i += c w Q,  g_bar_i += c w G d,  rho_bar_i += lambda_j c V_i S G / rho_i,  and per tile
//                sum lambda_i X_ij (-> delta_bar, c0_bar).  Written in SORTED order: dx4 = {x_bar, rho_bar}, gb4 = {g_bar, 0}.
constexpr int kDeltaState = 40;
template <int DIM, int GS, bool VARH, bool ADJ>
__global__ void __launch_bounds__(kPtMaxWarps * 32)
k_delta_term_tile(TileGeom tg, KPar kp, TileSizes ts, const float4 *__restrict__ pos4, const float4 *__restrict__ g4,
                  const float2 *__restrict__ lr, const uint32_t *__restrict__ cell_start,
                  const uint32_t *__restrict__ cell_end, const long long *__restrict__ row_ptr,
                  const uint16_t *__restrict__ col16, const uint32_t *__restrict__ perm, float *__restrict__ drho_io,
                  float4 *__restrict__ out4_io, float4 *__restrict__ dx4, float4 *__restrict__ gb4,
                  float *__restrict__ partial)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    size_t o = 0;
    float4 *A = reinterpret_cast<float4 *>(smem_raw + o); o += (size_t)ts.mcap * 16;
    float4 *B = reinterpret_cast<float4 *>(smem_raw + o); o += (size_t)ts.mcap * 16;
    float2 *C = reinterpret_cast<float2 *>(smem_raw + o); o += (size_t)ts.mcap * 8;
    uint32_t *rp = reinterpret_cast<uint32_t *>(smem_raw + o); o += (size_t)(ts.tcap + 4) * 4;
    uint16_t *selfq = reinterpret_cast<uint16_t *>(smem_raw + o); o += (size_t)ts.tcap * 2;
    o = (o + 15) & ~(size_t)15;
    uint16_t *ring = reinterpret_cast<uint16_t *>(smem_raw + o);
    __shared__ TileTab tt;
    __shared__ float red[kPtMaxWarps];
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) {
        if (ADJ && threadIdx.x == 0) partial[blockIdx.x] = 0.f;
        return;
    }
    stage_halo(tt, pos4, A, g4, B, nullptr, nullptr, ADJ ? lr : nullptr, C, nullptr, nullptr);
    stage_rows(tt, row_ptr, rp, selfq);
    cp_async_wait<0>();
    __syncthreads();
    stage_shift<DIM>(tt, A);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, gl = lane % GS;
    const HC hu = hc_uniform<DIM>(kp);
    const uint32_t row0 = tt.row0;
    float SX = 0.f;                                              // per lane: sum lambda_i V_j S G (c applied below)
    tile_row_passes<GS>(tt, rp, ring, ts.rb, col16, row_ptr[tt.row0],
        [&](uint32_t r, bool live, uint32_t b, uint32_t e_in, const uint16_t *idx) {
            const uint32_t qi = selfq[r];
            const uint32_t e = live ? e_in : b;
            const float4 pi = A[qi], gi = B[qi];
            float2 li = make_float2(0.f, 1.f);
            if (ADJ) li = C[qi];
            float acc = 0.f, xb[3] = {0.f, 0.f, 0.f}, gb[3] = {0.f, 0.f, 0.f}, rb = 0.f;
            for (uint32_t k = b + gl; k < e; k += GS) {
                const uint32_t j = idx[k];
                SPH_ASSERT(j < tt.M);
                const float4 pj = A[j], gj = B[j];
                const float d[3] = {pi.x - pj.x, pi.y - pj.y, DIM == 3 ? pi.z - pj.z : 0.f};
                const float r2 = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
                HC hc = hu;
                if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
                const float rr = fast_sqrt(r2);
                const float t = fmaxf(fmaf(-hc.invH, rr, 1.0f), 0.f);
                const float t2 = t * t, t4 = t2 * t2;
                const float G = hc.cG * fmaf(5.0f * hc.invH, rr, 1.0f) * (t4 * t);
                const float gs[3] = {gi.x + gj.x, gi.y + gj.y, DIM == 3 ? gi.z + gj.z : 0.f};
                const float S = fmaf(gs[2], d[2], fmaf(gs[1], d[1], gs[0] * d[0]));
                const float cc = VARH ? -0.5f * hc.kd : 1.0f;       // uniform h: the factor -delta l c0 is applied per row
                if (!ADJ) {
                    acc = fmaf(cc * gj.w, S * G, acc);
                } else {
                    const float2 lj = C[j];
                    const float K = hc.cK * t4;
                    const float w = cc * fmaf(li.x, gj.w, -(lj.x * gi.w));      // c (lambda_i V_j - lambda_j V_i)
                    const float SK = S * K;
#pragma unroll
                    for (int kk = 0; kk < DIM; ++kk) {
                        xb[kk] = fmaf(w, fmaf(gs[kk], G, SK * d[kk]), xb[kk]);
                        gb[kk] = fmaf(w * G, d[kk], gb[kk]);
                    }
                    rb = fmaf(cc * lj.x, S * G, rb);                            // x V_i / rho_i below
                    SX = fmaf(cc * li.x * gj.w, S * G, SX);
                }
            }
            const float cu = VARH ? 1.0f : -0.5f * hu.kd;
            if (!ADJ) {
                acc = group_sum<GS>(acc) * cu;
                if (gl == 0 && live) {
                    const uint32_t row = row0 + r;
                    if (out4_io) out4_io[row].w += acc;
                    else drho_io[perm[row]] += acc;
                }
            } else {
#pragma unroll
                for (int kk = 0; kk < DIM; ++kk) {
                    xb[kk] = group_sum<GS>(xb[kk]) * cu;
                    gb[kk] = group_sum<GS>(gb[kk]) * cu;
                }
                rb = group_sum<GS>(rb) * cu * gi.w / li.y;
                if (gl == 0 && live) {
                    const uint32_t row = row0 + r;
                    dx4[row] = make_float4(xb[0], xb[1], xb[2], rb);
                    gb4[row] = make_float4(gb[0], gb[1], gb[2], 0.f);
                }
            }
        });
    if (ADJ) {
        if (!VARH) SX *= -0.5f * hu.kd;
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) SX += __shfl_xor_sync(0xffffffffu, SX, o2);
        if (lane == 0) red[warp] = SX;
        __syncthreads();
        if (threadIdx.x == 0) {
            float v = 0.f;
            for (int w = 0; w < nwarps; ++w) v += red[w];
            partial[blockIdx.x] = v;
        }
    }
}

} // namespace

// ==========================================================================================
// host side
// ==========================================================================================
// lanes per row: measured on C3 (profiles/r01_c): RHS/density 16, VJP 8 (its row epilogue is heavier); 2D rows are short
static int tile_group(const sph_ctx *ctx, bool vjp)
{
    const int g = ctx->opt_group ? ctx->opt_group : (ctx->geom.dim == 3 && !vjp ? 16 : 8);
    return g == 4 ? 8 : g;
}

// threads per CTA, shared-memory carve-up and size for a pair kernel with `state_bytes` per halo particle, at most
// `max_warps` warps per CTA (its launch bound) and about `regs` registers per thread.  Picks the (CTAs per SM, warps per
// CTA) pair with the most resident warps that shared memory (228 KB per SM, 227 KB per CTA, 1 KB reserved per CTA) and
// the register file (64 K per SM, allocated per warp in units of 256) admit; ties go to more CTAs (measured on C3,
// profiles/r01_c: two co-resident CTAs beat one of twice the size -- their staging and epilogue phases overlap).
static void tile_launch_cfg(const sph_ctx *ctx, int state_bytes, int gs, size_t static_smem, int max_warps, int regs,
                            int *threads, TileSizes *ts, size_t *smem, uint32_t halo_max = 0)
{
    // halo_max: the most halo particles a CTA stages (default: those of a whole tile)
    ts->mcap = (int)(((halo_max ? halo_max : ctx->tile_Mmax) + 7u) & ~7u);
    ts->tcap = (int)((ctx->tile_Tmax + 7u) & ~7u);
    const double mean = ctx->n > 0 ? (double)ctx->nnz / (double)ctx->n : 1.0;
    int rb = (int)((32 / gs) * mean * 1.25) + 24;
    rb = (rb + 7) & ~7;
    if (rb < 64) rb = 64;
    ts->rb = rb;
    ts->bulk = ctx->opt_stage_bulk;
    ts->split = 1;
    const size_t fixed = (size_t)ts->mcap * state_bytes + (size_t)(ts->tcap + 4) * 4 + (size_t)ts->tcap * 2 + 16;
    const size_t sm_total = 233472, per_cta = 1024 + static_smem, cta_max = 232448 - static_smem;
    auto need = [&](int warps) { return fixed + (size_t)warps * 2 * rb * 2; };
    const int regs_warp = ((regs + 7) & ~7) * 32;
    int warps = 0, best = 0;
    if (ctx->opt_warps) {
        warps = ctx->opt_warps < max_warps ? ctx->opt_warps : max_warps;
    } else {
        const int cand[] = {24, 20, 16, 12, 10, 8, 6, 4};
        for (int c = 4; c >= 1; --c)
            for (int w : cand) {
                if (w > max_warps || need(w) > cta_max) continue;
                if ((size_t)c * (need(w) + per_cta) > sm_total || (long)c * w * regs_warp > 65536 || c * w > 64) continue;
                if (c * w > best) { best = c * w; warps = w; }
            }
    }
    if (warps == 0) warps = 2;
    while (warps > 2 && need(warps) > cta_max) warps >>= 1;           // tile_setup needs two warps
    if (need(warps) > cta_max) {                                   // last resort: a minimal ring (rows fall back to global reads)
        ts->rb = 8;
    }
    *threads = warps * 32;
    *smem = fixed + (size_t)warps * 2 * ts->rb * 2;
}

#define SPH_TILE_SMEM_ATTR(KERNEL, SMEM) \
    SPH_CUDA_TRY(cudaFuncSetAttribute(KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(SMEM)))

int sph_launch_density_tile(sph_ctx *ctx, const KPar &kp, const float *m_s, float *rho_out, const uint32_t *um,
                            const float *m_caller, cudaStream_t st)
{
    // um: device flag "all masses equal" of this call (or NULL: general variant only); both variants are enqueued and the
    // one whose turn it is not returns at once
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, false);
    for (int pass = 0; pass < (um ? 2 : 1); ++pass) {
        const bool UMv = um && pass == 0;
        int threads;
        TileSizes ts;
        size_t smem;
        // {x,y,z,h} (+ m) per halo particle; every variant compiles to <= 40 registers
        tile_launch_cfg(ctx, UMv ? 16 : 20, gs, sizeof(TileTab), kPtMaxWarps, 40, &threads, &ts, &smem);
        if (pass == 1) ctx->launches += 1;
#define SPH_DT_LAUNCH2(DIM, GS, VARH, UM)                                                                             \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_density_tile<DIM, GS, VARH, UM>), smem);                                                \
        k_density_tile<DIM, GS, VARH, UM><<<(unsigned)tg.ntiles, threads, smem, st>>>(                                \
            tg, kp, ts, ctx->pos_s.as<float4>(), m_s, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),   \
            ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->perm.as<uint32_t>(), rho_out, um, m_caller); \
    } while (0)
#define SPH_DT_LAUNCH(DIM, GS, VARH)                                                                                  \
    do {                                                                                                              \
        if (UMv) SPH_DT_LAUNCH2(DIM, GS, VARH, true); else SPH_DT_LAUNCH2(DIM, GS, VARH, false);                      \
    } while (0)
#define SPH_DT_GS(GS)                                                                                     \
    do {                                                                                                  \
        if (kp.dim == 3) { if (kp.uniform_h) SPH_DT_LAUNCH(3, GS, false); else SPH_DT_LAUNCH(3, GS, true); } \
        else { if (kp.uniform_h) SPH_DT_LAUNCH(2, GS, false); else SPH_DT_LAUNCH(2, GS, true); }             \
    } while (0)
        switch (gs) {
        case 16: SPH_DT_GS(16); break;
        case 32: SPH_DT_GS(32); break;
        default: SPH_DT_GS(8); break;
        }
#undef SPH_DT_GS
#undef SPH_DT_LAUNCH
#undef SPH_DT_LAUNCH2
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int sph_launch_density_vjp_tile(sph_ctx *ctx, const KPar &kp, const float2 *mr_s, float *x_bar, float *m_bar,
                                cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, false);
    int threads;
    TileSizes ts;
    size_t smem;
    tile_launch_cfg(ctx, kp.dim == 3 ? 40 : 32, gs, sizeof(TileTab), kPtMaxWarps, 64, &threads, &ts, &smem);   // carve-up of SmemMap
#define SPH_DVT_LAUNCH(DIM, GS, VARH)                                                                                 \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_density_vjp_tile<DIM, GS, VARH>), smem);                                                \
        k_density_vjp_tile<DIM, GS, VARH><<<(unsigned)tg.ntiles, threads, smem, st>>>(                                \
            tg, kp, ts, ctx->pos_s.as<float4>(), mr_s, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),  \
            ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->perm.as<uint32_t>(), x_bar, m_bar);         \
    } while (0)
#define SPH_DVT_GS(GS)                                                                                      \
    do {                                                                                                    \
        if (kp.dim == 3) { if (kp.uniform_h) SPH_DVT_LAUNCH(3, GS, false); else SPH_DVT_LAUNCH(3, GS, true); } \
        else { if (kp.uniform_h) SPH_DVT_LAUNCH(2, GS, false); else SPH_DVT_LAUNCH(2, GS, true); }             \
    } while (0)
    switch (gs) {
    case 16: SPH_DVT_GS(16); break;
    case 32: SPH_DVT_GS(32); break;
    default: SPH_DVT_GS(8); break;
    }
#undef SPH_DVT_GS
#undef SPH_DVT_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int sph_launch_renorm_tile(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float2 *va_s, float4 *mom, cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, false);
    int threads;
    TileSizes ts;
    size_t smem;
    tile_launch_cfg(ctx, kp.dim == 3 ? 40 : 32, gs, sizeof(TileTab), kPtMaxWarps, 64, &threads, &ts, &smem);   // carve-up of SmemMap
#define SPH_RNT_LAUNCH(DIM, GS, VARH)                                                                                 \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_renorm_tile<DIM, GS, VARH>), smem);                                                     \
        k_renorm_tile<DIM, GS, VARH><<<(unsigned)tg.ntiles, threads, smem, st>>>(                                     \
            tg, kp, ts, pos4, va_s, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),                     \
            ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), mom);                                            \
    } while (0)
#define SPH_RNT_GS(GS)                                                                                      \
    do {                                                                                                    \
        if (kp.dim == 3) { if (kp.uniform_h) SPH_RNT_LAUNCH(3, GS, false); else SPH_RNT_LAUNCH(3, GS, true); } \
        else { if (kp.uniform_h) SPH_RNT_LAUNCH(2, GS, false); else SPH_RNT_LAUNCH(2, GS, true); }             \
    } while (0)
    switch (gs) {
    case 16: SPH_RNT_GS(16); break;
    case 32: SPH_RNT_GS(32); break;
    default: SPH_RNT_GS(8); break;
    }
#undef SPH_RNT_GS
#undef SPH_RNT_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int sph_launch_renorm_vjp_tile(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *rb, const float4 *rc,
                               const float2 *rd, const float *re, const uint32_t *perm, float *x_bar, float *vol_bar,
                               float *A_bar, cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, true);
    int threads;
    TileSizes ts;
    size_t smem;
    tile_launch_cfg(ctx, kp.dim == 3 ? 60 : 44, gs, sizeof(TileTab), kPtMaxWarps, 96, &threads, &ts, &smem);   // carve-up of k_renorm_vjp_tile
#define SPH_RNVT_LAUNCH(DIM, GS, VARH)                                                                                \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_renorm_vjp_tile<DIM, GS, VARH>), smem);                                                 \
        k_renorm_vjp_tile<DIM, GS, VARH><<<(unsigned)tg.ntiles, threads, smem, st>>>(                                 \
            tg, kp, ts, pos4, rb, rc, rd, re, ctx->cell_start.as<uint32_t>(),                                         \
            ctx->cell_end.as<uint32_t>(), ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(),                    \
            perm, x_bar, vol_bar, A_bar);                                                         \
    } while (0)
#define SPH_RNVT_GS(GS)                                                                                       \
    do {                                                                                                      \
        if (kp.dim == 3) { if (kp.uniform_h) SPH_RNVT_LAUNCH(3, GS, false); else SPH_RNVT_LAUNCH(3, GS, true); } \
        else { if (kp.uniform_h) SPH_RNVT_LAUNCH(2, GS, false); else SPH_RNVT_LAUNCH(2, GS, true); }             \
    } while (0)
    switch (gs) {
    case 16: SPH_RNVT_GS(16); break;
    case 32: SPH_RNVT_GS(32); break;
    default: SPH_RNVT_GS(8); break;
    }
#undef SPH_RNVT_GS
#undef SPH_RNVT_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

static int launch_grad_sum_tile(sph_ctx *ctx, const KPar &kp, const float *a_s, const float4 *ga_s, float *v_out,
                                float *a_out, bool vjp, cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, false);
    int threads;
    TileSizes ts;
    size_t smem;
    tile_launch_cfg(ctx, kp.dim == 3 ? 40 : 32, gs, sizeof(TileTab), kPtMaxWarps, 64, &threads, &ts, &smem);   // carve-up of SmemMap
#define SPH_GT_LAUNCH(DIM, GS, VARH, VJP)                                                                             \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_grad_sum_tile<DIM, GS, VARH, VJP>), smem);                                              \
        k_grad_sum_tile<DIM, GS, VARH, VJP><<<(unsigned)tg.ntiles, threads, smem, st>>>(                              \
            tg, kp, ts, ctx->pos_override ? ctx->pos_override : ctx->pos_s.as<float4>(), a_s, ga_s,                   \
            ctx->cell_start.as<uint32_t>(),                                                                           \
            ctx->cell_end.as<uint32_t>(), ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(),                    \
            ctx->perm.as<uint32_t>(), v_out, a_out);                                                                  \
    } while (0)
#define SPH_GT_GS(GS)                                                                                                 \
    do {                                                                                                              \
        if (kp.dim == 3) {                                                                                            \
            if (kp.uniform_h) { if (vjp) SPH_GT_LAUNCH(3, GS, false, true); else SPH_GT_LAUNCH(3, GS, false, false); } \
            else { if (vjp) SPH_GT_LAUNCH(3, GS, true, true); else SPH_GT_LAUNCH(3, GS, true, false); }                \
        } else {                                                                                                      \
            if (kp.uniform_h) { if (vjp) SPH_GT_LAUNCH(2, GS, false, true); else SPH_GT_LAUNCH(2, GS, false, false); } \
            else { if (vjp) SPH_GT_LAUNCH(2, GS, true, true); else SPH_GT_LAUNCH(2, GS, true, false); }                \
        }                                                                                                             \
    } while (0)
    switch (gs) {
    case 16: SPH_GT_GS(16); break;
    case 32: SPH_GT_GS(32); break;
    default: SPH_GT_GS(8); break;
    }
#undef SPH_GT_GS
#undef SPH_GT_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int sph_launch_grad_sum_tile(sph_ctx *ctx, const KPar &kp, const float *a_s, float *g_out, cudaStream_t st)
{
    return launch_grad_sum_tile(ctx, kp, a_s, nullptr, g_out, nullptr, false, st);
}

int sph_launch_grad_sum_vjp_tile(sph_ctx *ctx, const KPar &kp, const float4 *ga_s, float *x_bar, float *a_bar,
                                 cudaStream_t st)
{
    return launch_grad_sum_tile(ctx, kp, nullptr, ga_s, x_bar, a_bar, true, st);
}

// Both pair kernels come in a general variant and (3D, uniform h) a uniform-mass one that gathers 32 / 48 instead of
// 40 / 56 bytes per pair.  Whether the masses are uniform is known on the device only (sph_um_flag, written by the pack
// kernel of this call on the same stream), so both variants are enqueued, each with its own shared-memory carve-up, and
// the one whose turn it is not returns in its first instruction.
int sph_launch_rhs_tile(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                        const uint8_t *kind_s, float *drho, float *acc, float4 *out4, cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, false);
    const bool sorted = out4 != nullptr;
    const bool dual = kp.dim == 3 && kp.uniform_h && !ctx->opt_no_um;
    const uint32_t *um = dual ? sph_um_flag(ctx) : nullptr;
    for (int pass = 0; pass < (dual ? 2 : 1); ++pass) {
        const bool UMv = dual && pass == 0;
        int threads;
        TileSizes ts;
        size_t smem;
        const unsigned grid = (unsigned)tg.ntiles;
        tile_launch_cfg(ctx, kp.dim == 3 ? (UMv ? 32 : 40) : 32, gs, sizeof(TileTab), kPtMaxWarps, 64, &threads, &ts, &smem);
        if (pass == 1) ctx->launches += 1;                     // the second variant is a launch too
#define SPH_RT_LAUNCH2(DIM, GS, VARH, SORTED, F1, UM)                                                                \
    do {                                                                                                             \
        SPH_TILE_SMEM_ATTR((k_rhs_tile<DIM, GS, VARH, SORTED, F1, UM>), smem);                                       \
        k_rhs_tile<DIM, GS, VARH, SORTED, F1, UM><<<grid, threads, smem, st>>>(                                      \
            tg, kp, ts, s0, s1, s2, kind_s, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),            \
            ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->perm.as<uint32_t>(), drho, acc, out4, um); \
    } while (0)
#define SPH_RT_LAUNCH1(DIM, GS, VARH, SORTED, F1)                                                                    \
    do {                                                                                                             \
        if (DIM == 3 && !VARH && UMv) SPH_RT_LAUNCH2(3, GS, false, SORTED, F1, true);                                \
        else SPH_RT_LAUNCH2(DIM, GS, VARH, SORTED, F1, false);                                                       \
    } while (0)
#define SPH_RT_LAUNCH(DIM, GS, VARH, SORTED)                                                                         \
    do {                                                                                                             \
        if (kp.form == 0) SPH_RT_LAUNCH1(DIM, GS, VARH, SORTED, false); else SPH_RT_LAUNCH1(DIM, GS, VARH, SORTED, true); \
    } while (0)
#define SPH_RT_GS(GS)                                                                                                   \
    do {                                                                                                                \
        if (kp.dim == 3) {                                                                                              \
            if (kp.uniform_h) { if (sorted) SPH_RT_LAUNCH(3, GS, false, true); else SPH_RT_LAUNCH(3, GS, false, false); } \
            else { if (sorted) SPH_RT_LAUNCH(3, GS, true, true); else SPH_RT_LAUNCH(3, GS, true, false); }                \
        } else {                                                                                                        \
            if (kp.uniform_h) { if (sorted) SPH_RT_LAUNCH(2, GS, false, true); else SPH_RT_LAUNCH(2, GS, false, false); } \
            else { if (sorted) SPH_RT_LAUNCH(2, GS, true, true); else SPH_RT_LAUNCH(2, GS, true, false); }                \
        }                                                                                                               \
    } while (0)
        switch (gs) {
        case 16: SPH_RT_GS(16); break;
        case 32: SPH_RT_GS(32); break;
        default: SPH_RT_GS(8); break;
        }
#undef SPH_RT_GS
#undef SPH_RT_LAUNCH
#undef SPH_RT_LAUNCH1
#undef SPH_RT_LAUNCH2
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

// CTAs per tile of k_vjp_tile: 2 in 3D on 2x2x2-cell tiles (each CTA takes one z-layer of the block)
int sph_vjp_tile_split(const sph_ctx *ctx, const KPar &kp)
{
    return (ctx->opt_vjp_split && kp.dim == 3 && ctx->tg.B == 2 && ctx->tile_Mhalf > 0) ? 2 : 1;
}

int sph_launch_vjp_tile(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                        const float4 *cot, const float4 *eos, float *xb, float *vb, float *rb, float4 *xb4, float4 *vb4,
                        float *partials, cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, true);
    const bool sorted = xb4 != nullptr;
    const bool dual = kp.dim == 3 && kp.uniform_h && !ctx->opt_no_um;
    const uint32_t *um = dual ? sph_um_flag(ctx) : nullptr;
    const int split = sph_vjp_tile_split(ctx, kp);
    const unsigned grid = (unsigned)tg.ntiles * (unsigned)split;
    for (int pass = 0; pass < (dual ? 2 : 1); ++pass) {
        const bool UMv = dual && pass == 0;
        int threads;
        TileSizes ts;
        size_t smem;
        tile_launch_cfg(ctx, kp.dim == 3 ? (UMv ? 48 : 56) : 48, gs, sizeof(TileTab) + kVjpMaxWarps * kNPartT * 4, kVjpMaxWarps, 80, &threads,
                        &ts, &smem, split == 2 ? ctx->tile_Mhalf : 0u);
        ts.split = split;
        if (pass == 1) ctx->launches += 1;
#define SPH_VT_LAUNCH2(DIM, GS, VARH, SORTED, F1, UM)                                                                 \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_vjp_tile<DIM, GS, VARH, SORTED, F1, UM>), smem);                                        \
        k_vjp_tile<DIM, GS, VARH, SORTED, F1, UM><<<grid, threads, smem, st>>>(                                       \
            tg, kp, ts, s0, s1, s2, cot, eos, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),           \
            ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->perm.as<uint32_t>(), xb, vb, rb, xb4, vb4,  \
            partials, um);                                                                                            \
    } while (0)
#define SPH_VT_LAUNCH1(DIM, GS, VARH, SORTED, F1)                                                                     \
    do {                                                                                                              \
        if (DIM == 3 && !VARH && UMv) SPH_VT_LAUNCH2(3, GS, false, SORTED, F1, true);                                 \
        else SPH_VT_LAUNCH2(DIM, GS, VARH, SORTED, F1, false);                                                        \
    } while (0)
#define SPH_VT_LAUNCH(DIM, GS, VARH, SORTED)                                                                          \
    do {                                                                                                              \
        if (kp.form == 0) SPH_VT_LAUNCH1(DIM, GS, VARH, SORTED, false); else SPH_VT_LAUNCH1(DIM, GS, VARH, SORTED, true); \
    } while (0)
#define SPH_VT_GS(GS)                                                                                                   \
    do {                                                                                                                \
        if (kp.dim == 3) {                                                                                              \
            if (kp.uniform_h) { if (sorted) SPH_VT_LAUNCH(3, GS, false, true); else SPH_VT_LAUNCH(3, GS, false, false); } \
            else { if (sorted) SPH_VT_LAUNCH(3, GS, true, true); else SPH_VT_LAUNCH(3, GS, true, false); }                \
        } else {                                                                                                        \
            if (kp.uniform_h) { if (sorted) SPH_VT_LAUNCH(2, GS, false, true); else SPH_VT_LAUNCH(2, GS, false, false); } \
            else { if (sorted) SPH_VT_LAUNCH(2, GS, true, true); else SPH_VT_LAUNCH(2, GS, true, false); }                \
        }                                                                                                               \
    } while (0)
        switch (gs) {
        case 16: SPH_VT_GS(16); break;
        case 32: SPH_VT_GS(32); break;
        default: SPH_VT_GS(8); break;
        }
#undef SPH_VT_GS
#undef SPH_VT_LAUNCH
#undef SPH_VT_LAUNCH1
#undef SPH_VT_LAUNCH2
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

// delta-term of [43] (tile layout); see k_delta_term_tile.  pos4/g4/lr: sorted arrays of the current state.
int sph_launch_delta_term_tile(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *g4, const float2 *lr,
                               bool adjoint, float *drho_io, float4 *out4_io, float4 *dx4, float4 *gb4, float *partial,
                               cudaStream_t st)
{
    const TileGeom &tg = ctx->tg;
    const int gs = tile_group(ctx, false);
    int threads;
    TileSizes ts;
    size_t smem;
    tile_launch_cfg(ctx, kDeltaState, gs, sizeof(TileTab) + kPtMaxWarps * 4, kPtMaxWarps, 64, &threads, &ts, &smem);
#define SPH_DLT_LAUNCH(DIM, GS, VARH, ADJ)                                                                            \
    do {                                                                                                              \
        SPH_TILE_SMEM_ATTR((k_delta_term_tile<DIM, GS, VARH, ADJ>), smem);                                            \
        k_delta_term_tile<DIM, GS, VARH, ADJ><<<(unsigned)tg.ntiles, threads, smem, st>>>(                            \
            tg, kp, ts, pos4, g4, lr, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),                   \
            ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->perm.as<uint32_t>(), drho_io, out4_io, dx4, \
            gb4, partial);                                                                                            \
    } while (0)
#define SPH_DLT_GS(GS)                                                                                                \
    do {                                                                                                              \
        if (kp.dim == 3) {                                                                                            \
            if (kp.uniform_h) { if (adjoint) SPH_DLT_LAUNCH(3, GS, false, true); else SPH_DLT_LAUNCH(3, GS, false, false); } \
            else { if (adjoint) SPH_DLT_LAUNCH(3, GS, true, true); else SPH_DLT_LAUNCH(3, GS, true, false); }           \
        } else {                                                                                                      \
            if (kp.uniform_h) { if (adjoint) SPH_DLT_LAUNCH(2, GS, false, true); else SPH_DLT_LAUNCH(2, GS, false, false); } \
            else { if (adjoint) SPH_DLT_LAUNCH(2, GS, true, true); else SPH_DLT_LAUNCH(2, GS, true, false); }           \
        }                                                                                                             \
    } while (0)
    switch (gs) {
    case 16: SPH_DLT_GS(16); break;
    default: SPH_DLT_GS(8); break;
    }
#undef SPH_DLT_GS
#undef SPH_DLT_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

#ifdef SPH_BOUNDS
unsigned int sph_bounds_read_pairs_tile()
{
    unsigned int v = 0;
    cudaMemcpyFromSymbol(&v, sph_bounds_count, sizeof(v));
    return v;
}
#endif
