// sph_neighbors_tile.cu -- steps N5/N7 of SURVEY.md 8(a) on the cell-block decomposition of sph_tiles.cuh:
// count and fill of TILE-LOCAL compact lists (uint16 halo-linear indices), PAPER.md:558 (adjacent-cell query),
// PAPER.md:163 (pair list), PAPER.md:167 (radius max{h_i,h_j}).
//
// Count (k_nb_tile<FILL=0>): one CTA per tile.  The halo positions are staged in shared memory once.  A warp takes 32
// rows OF ONE CELL, one row per lane: all lanes walk the same candidate sequence, so every candidate is ONE broadcast
// shared-memory load and 8-9 instructions for 32 row-candidate tests (the first path of this round spent 110 per 32):
// the verdict is the sign bit of r2 - Hs2, funnel-shifted into a per-lane 32-candidate mask; the binary64 predicate of
// reading R3 runs only for blocks whose closest call falls inside the fp32 uncertainty band.  The count of a row is the
// popcount of its masks; the masks are kept (coalesced, [item][word][lane]).
// Fill (k_nb_expand): no distance is computed twice.  Same work items; a lane expands the masks of its row in candidate
// order (cells in z,y,x order, ascending sorted index inside a cell) into a per-warp shared-memory image of the warp's
// contiguous col16 segment (rows of a cell are contiguous in the sorted order, so their list segments are too), which
// is then flushed coalesced.  k_nb_tile<FILL=1> is the variant that repeats the tests (no mask buffer).
// Deterministic: fixed candidate order, no atomics.
#include "sph_internal.cuh"
#include "sph_tiles.cuh"
#include "sph_search.cuh"

#include <math.h>

namespace {

constexpr int kNbWarps = 8;
constexpr uint32_t kWqCap = 96;    // mask words per row handled by the fast expansion

struct RowCtx {
    float4 pi;         // own position (+h)
    float Hs2, tol;    // uniform h: thresholds of the fp32 test
    uint32_t n;        // hits so far
};

// fp32 test of one candidate: shifts the verdict (sign of r2 - Hs2) into the mask and tracks how close to the
// threshold the block came.  9 instructions per candidate when h is uniform.
template <int DIM, bool VARH>
__device__ __forceinline__ void nb_test(const RowCtx &rc, const float4 &pj, const SearchPar &sp, bool seam, uint32_t &m,
                                        float &amin)
{
    const float d0 = rc.pi.x - pj.x, d1 = rc.pi.y - pj.y, d2 = DIM == 3 ? rc.pi.z - pj.z : 0.f;
    // diff = r2 - Hs2 with the subtraction folded into the FMA chain (one instruction less; its rounding error,
    // < 2^-22 Hs2, is covered by the 2^-19 band like that of r2 itself)
    if (VARH) {
        const float Hs = __fmul_rn(sp.scale, fmaxf(rc.pi.w, pj.w));
        const float Hs2 = Hs * Hs;
        const float tol = sp.band * (seam ? fmaf(Hs, sp.Lmax, Hs2) : Hs2);
        const float diff = fmaf(d2, d2, fmaf(d1, d1, fmaf(d0, d0, -Hs2)));
        m = __funnelshift_l(__float_as_uint(diff), m, 1);       // m = (m << 1) | (diff < 0)
        amin = fminf(amin, fabsf(diff) - tol);
    } else {
        const float diff = fmaf(d2, d2, fmaf(d1, d1, fmaf(d0, d0, -rc.Hs2)));
        m = __funnelshift_l(__float_as_uint(diff), m, 1);
        amin = fminf(amin, fabsf(diff));
    }
}

// the same test with the "too close to call" band resolved by the binary64 predicate (reading R3)
template <int DIM, bool VARH>
__device__ __forceinline__ bool nb_test_exact(const RowCtx &rc, const float4 &pj, const SearchPar &sp, bool seam,
                                              uint32_t q, const TileTab &tt, const float4 *__restrict__ pos_s,
                                              const GridGeom &gg)
{
    const float d0 = rc.pi.x - pj.x, d1 = rc.pi.y - pj.y, d2 = DIM == 3 ? rc.pi.z - pj.z : 0.f;
    float Hs2 = rc.Hs2, tol = rc.tol, Hs = sp.Hs_u;
    if (VARH) {
        Hs = __fmul_rn(sp.scale, fmaxf(rc.pi.w, pj.w));
        Hs2 = Hs * Hs;
        tol = sp.band * (seam ? fmaf(Hs, sp.Lmax, Hs2) : Hs2);
    }
    const float diff = fmaf(d2, d2, fmaf(d1, d1, fmaf(d0, d0, -Hs2)));
    bool hit = diff < 0.f;
    if (fabsf(diff) <= tol) hit = pred_exact(rc.pi, pos_s[tile_q_to_sorted(tt, q)], Hs, gg);
    return hit;
}

// Hit mask of the nq <= 32 candidates q .. q+nq-1 for this lane's row: candidate u at bit nq-1-u.
template <int DIM, bool VARH, bool FULL>
__device__ __forceinline__ uint32_t nb_mask(const RowCtx &rc, const float4 *__restrict__ cand, uint32_t q, int nq,
                                            const SearchPar &sp, bool seam, const TileTab &tt,
                                            const float4 *__restrict__ pos_s, const GridGeom &gg)
{
    uint32_t m = 0;
    float amin = 3.0e38f;
    if (FULL) {
#pragma unroll
        for (int u = 0; u < 32; ++u) nb_test<DIM, VARH>(rc, cand[q + u], sp, seam, m, amin);
    } else {
#pragma unroll 4
        for (int u = 0; u < nq; ++u) nb_test<DIM, VARH>(rc, cand[q + u], sp, seam, m, amin);
    }
    if (amin <= (VARH ? 0.f : rc.tol)) {              // rare (except on exact lattices): redo the block exactly
        m = 0;
        for (int u = 0; u < nq; ++u)
            m = (m << 1) | (nb_test_exact<DIM, VARH>(rc, cand[q + u], sp, seam, q + u, tt, pos_s, gg) ? 1u : 0u);
    }
    return m;
}

// mask words per row of the cell at halo slot sl: one per 32 candidates of each of its 3^(d-1) x-runs
template <int DIM>
__device__ __forceinline__ uint32_t cell_words(const TileTab &tt, const int sl[3])
{
    uint32_t w = 0;
    const int zlo = DIM == 3 ? -1 : 0, zhi = DIM == 3 ? 1 : 0;
    for (int dz = zlo; dz <= zhi; ++dz) {
        const int sz = sl[2] + dz;
        if (DIM == 3 && (sz < 0 || sz >= tt.ext[2])) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            const int sy = sl[1] + dy;
            if (sy < 0 || sy >= tt.ext[1]) continue;
            const int rowbase = tt.ext[0] * (sy + tt.ext[1] * sz);
            const int xa = max(sl[0] - 1, 0), xb = min(sl[0] + 1, tt.ext[0] - 1);
            w += (tt.h_off[rowbase + xb + 1] - tt.h_off[rowbase + xa] + 31u) >> 5;
        }
    }
    return w;
}

// `dst`: FILL only -- where this lane's hits go (shared-memory image or global col16), indexed by rc.n
// `maskp` (count pass, may be null): this lane's column of the item's mask block; word w of the row at maskp[32 w]
template <int DIM, bool FILL, bool VARH, class DstT>
__device__ __forceinline__ void nb_rows(RowCtx &rc, const float4 *__restrict__ cand, const int sl[3], const SearchPar &sp,
                                        bool seam, const TileTab &tt, const float4 *__restrict__ pos_s,
                                        const GridGeom &gg, DstT dst, uint32_t *__restrict__ maskp = nullptr)
{
    const int zlo = DIM == 3 ? -1 : 0, zhi = DIM == 3 ? 1 : 0;
    for (int dz = zlo; dz <= zhi; ++dz) {
        const int sz = sl[2] + dz;
        if (DIM == 3 && (sz < 0 || sz >= tt.ext[2])) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            const int sy = sl[1] + dy;
            if (sy < 0 || sy >= tt.ext[1]) continue;
            const int rowbase = tt.ext[0] * (sy + tt.ext[1] * sz);
            const int xa = max(sl[0] - 1, 0), xb = min(sl[0] + 1, tt.ext[0] - 1);
            const uint32_t q0 = tt.h_off[rowbase + xa], q1 = tt.h_off[rowbase + xb + 1];
            for (uint32_t q = q0; q < q1; q += 32) {
                const int nq = min(32u, q1 - q);
                uint32_t m = nq == 32 ? nb_mask<DIM, VARH, true>(rc, cand, q, 32, sp, seam, tt, pos_s, gg)
                                      : nb_mask<DIM, VARH, false>(rc, cand, q, nq, sp, seam, tt, pos_s, gg);
                if (FILL) {
                    const uint32_t qtop = q + (uint32_t)nq - 1u;      // candidate of bit 0
                    while (m) {                                         // ascending candidate order = descending bits
                        const int hb = 31 - __clz(m);
                        m ^= 1u << hb;
                        dst[rc.n++] = (uint16_t)(qtop - (uint32_t)hb);
                    }
                } else {
                    rc.n += __popc(m);
                    if (maskp) {
                        *maskp = m;
                        maskp += 32;
                    }
                }
            }
        }
    }
}

template <int DIM, bool FILL, bool VARH>
__global__ void __launch_bounds__(kNbWarps * 32)
k_nb_tile(TileGeom tg, GridGeom gg, SearchPar sp, int mcap, int wcap, const float4 *__restrict__ pos_s,
          const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end, uint32_t *__restrict__ cnt,
          const long long *__restrict__ row_ptr, uint16_t *__restrict__ col16, uint32_t *__restrict__ maskbuf,
          const long long *__restrict__ tile_mask_base)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *cand = reinterpret_cast<float4 *>(smem_raw);
    __shared__ TileTab tt;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    bool seam = false;
#pragma unroll
    for (int k = 0; k < DIM; ++k)
        if (tg.periodic[k] && (tt.hs[k] < 0 || tt.hs[k] + tt.ext[k] > tg.ncell[k])) seam = true;

    // ---- stage the halo positions (shifted across periodic seams)
    for (int hc = warp; hc < tt.nh; hc += kNbWarps) {
        const uint32_t o0 = tt.h_off[hc], o1 = tt.h_off[hc + 1];
        if (o1 == o0) continue;
        float sh[3];
        tile_cell_shift<DIM>(tg, tt, hc, sh);
        const uint32_t gs = tt.h_start[hc];
        for (uint32_t q = o0 + lane; q < o1; q += 32) {
            float4 pj = pos_s[gs + (q - o0)];
            pj.x += sh[0];
            pj.y += sh[1];
            if (DIM == 3) pj.z += sh[2];
            cand[q] = pj;
        }
    }
    __syncthreads();

    uint16_t *wbuf = reinterpret_cast<uint16_t *>(smem_raw + (size_t)mcap * sizeof(float4)) + (size_t)warp * wcap;
    // ---- work items: (target cell, chunk of 32 rows), dealt round-robin to the warps
    int item = 0;
    long long mask_off = maskbuf ? tile_mask_base[blockIdx.x] : 0;   // start of the next item's mask block
    for (int tc = 0; tc < tt.nt; ++tc) {
        const uint32_t nrow = tt.t_off[tc + 1] - tt.t_off[tc];
        const int hc_i = tt.t_cell[tc];
        const int sl[3] = {hc_i % tt.ext[0], (hc_i / tt.ext[0]) % tt.ext[1], hc_i / (tt.ext[0] * tt.ext[1])};
        const uint32_t item_words = (!FILL && maskbuf && nrow) ? 32u * cell_words<DIM>(tt, sl) : 0u;
        for (uint32_t c0 = 0; c0 < nrow; c0 += 32, ++item, mask_off += item_words) {
            if (item % kNbWarps != warp) continue;
            const uint32_t nact = min(32u, nrow - c0);
            const bool active = (uint32_t)lane < nact;
            const uint32_t local = c0 + (active ? lane : 0);
            const uint32_t row = tt.h_start[hc_i] + local;
            RowCtx rc;
            rc.pi = cand[tt.h_off[hc_i] + local];          // target cells are never shifted
            rc.Hs2 = sp.Hs_u * sp.Hs_u;
            rc.tol = sp.band * (seam ? fmaf(sp.Hs_u, sp.Lmax, rc.Hs2) : rc.Hs2);
            rc.n = 0;
            if (!FILL) {
                nb_rows<DIM, false, VARH>(rc, cand, sl, sp, seam, tt, pos_s, gg, (uint16_t *)nullptr,
                                          maskbuf ? maskbuf + mask_off + lane : nullptr);
                if (active) cnt[row] = rc.n;
            } else {
                const uint32_t row_first = tt.h_start[hc_i] + c0;
                const long long seg0 = row_ptr[row_first], seg1 = row_ptr[row_first + nact];
                const long long mine = row_ptr[row];
                const uint32_t total = (uint32_t)(seg1 - seg0);
                if (total <= (uint32_t)wcap) {
                    // inactive lanes duplicate lane 0 and write the same values to the same places
                    nb_rows<DIM, true, VARH>(rc, cand, sl, sp, seam, tt, pos_s, gg, wbuf + (uint32_t)(mine - seg0));
                    __syncwarp();
                    uint16_t *out = col16 + seg0;
                    for (uint32_t k = lane; k < total; k += 32) out[k] = wbuf[k];
                    __syncwarp();
                } else {
                    nb_rows<DIM, true, VARH>(rc, cand, sl, sp, seam, tt, pos_s, gg, col16 + mine);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------- masks -> lists
// mask words of every tile (same item enumeration as k_nb_tile): words[tile] = sum over items of 32 * cell_words
template <int DIM>
__global__ void __launch_bounds__(64)
k_tile_words(TileGeom tg, const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
             uint32_t *__restrict__ words, uint32_t *__restrict__ wmax_out)
{
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (threadIdx.x >= 32) return;
    uint32_t w = 0;
    const int tc = threadIdx.x;
    if (tc < tt.nt) {
        const uint32_t nrow = tt.t_off[tc + 1] - tt.t_off[tc];
        const int hc_i = tt.t_cell[tc];
        const int sl[3] = {hc_i % tt.ext[0], (hc_i / tt.ext[0]) % tt.ext[1], hc_i / (tt.ext[0] * tt.ext[1])};
        uint32_t cw = 0;
        if (nrow) {
            cw = cell_words<DIM>(tt, sl);
            w = ((nrow + 31u) >> 5) * 32u * cw;
        }
        cw = __reduce_max_sync(0xffffffffu, cw);
        if (threadIdx.x == 0 && cw > *(volatile uint32_t *)wmax_out) atomicMax(wmax_out, cw);
    } else {
        (void)__reduce_max_sync(0xffffffffu, 0u);
    }
    w = __reduce_add_sync(0xffffffffu, w);
    if (threadIdx.x == 0) words[blockIdx.x] = w;
}

// N7 from the hit masks of the count pass: no distance test is repeated.  Same work items as k_nb_tile (32 rows of one
// cell per warp, one row per lane); every lane expands its own mask words in candidate order into the warp's
// shared-memory image of its contiguous col16 segment, which is flushed coalesced.
template <int DIM>
__global__ void __launch_bounds__(kNbWarps * 32)
k_nb_expand(TileGeom tg, int wcap, int wbcap, const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
            const long long *__restrict__ row_ptr, uint16_t *__restrict__ col16, const uint32_t *__restrict__ maskbuf,
            const long long *__restrict__ tile_mask_base)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ TileTab tt;
    __shared__ uint16_t wqtab[kNbWarps][kWqCap];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    const int nwarps = blockDim.x >> 5;
    // per warp: image of its col16 segment (wcap entries) and the mask block of its item (wbcap words x 32 lanes)
    uint16_t *wbuf = reinterpret_cast<uint16_t *>(smem_raw) + (size_t)warp * wcap;
    uint32_t *mblk = reinterpret_cast<uint32_t *>(smem_raw + (size_t)nwarps * wcap * 2) + (size_t)warp * wbcap * 32;
    // word table of the warp: the static one, or (rows with more than kWqCap mask words: dense cells, config 4) a
    // dynamic one of wbcap entries behind the mask blocks
    const uint32_t wqcap = (uint32_t)wbcap > kWqCap ? (uint32_t)wbcap : kWqCap;
    uint16_t *wq_dyn = reinterpret_cast<uint16_t *>(smem_raw + (size_t)nwarps * ((size_t)wcap * 2 + (size_t)wbcap * 128)) +
                       (size_t)warp * wbcap;
    int item = 0;
    long long mask_off = tile_mask_base[blockIdx.x];
    for (int tc = 0; tc < tt.nt; ++tc) {
        const uint32_t nrow = tt.t_off[tc + 1] - tt.t_off[tc];
        const int hc_i = tt.t_cell[tc];
        const int sl[3] = {hc_i % tt.ext[0], (hc_i / tt.ext[0]) % tt.ext[1], hc_i / (tt.ext[0] * tt.ext[1])};
        const uint32_t item_words = nrow ? 32u * cell_words<DIM>(tt, sl) : 0u;
        for (uint32_t c0 = 0; c0 < nrow; c0 += 32, ++item, mask_off += item_words) {
            if (item % nwarps != warp) continue;
            const uint32_t nact = min(32u, nrow - c0);
            const bool active = (uint32_t)lane < nact;
            const uint32_t row_first = tt.h_start[hc_i] + c0;
            const uint32_t row = row_first + (active ? lane : 0);
            const long long seg0 = row_ptr[row_first], seg1 = row_ptr[row_first + nact];
            const long long mine = row_ptr[row];
            const uint32_t total = (uint32_t)(seg1 - seg0);
            const bool staged = total <= (uint32_t)wcap;
            // inactive lanes duplicate lane 0: same masks, same values to the same places
            const uint32_t *mp = maskbuf + mask_off + (active ? lane : 0);
            uint16_t *dst_s = wbuf + (uint32_t)(mine - seg0);
            uint16_t *dst_g = col16 + mine;
            // the item's mask block into shared memory with cp.async (all W x 128 B in flight at once, overlapped
            // with the table build below; a plain load/store loop exposes the global latency once per word)
            const uint32_t Wi = item_words >> 5;
            if (Wi <= wqcap && Wi <= (uint32_t)wbcap) {
                const uint32_t *src = maskbuf + mask_off + lane;
                const uint32_t dsts = (uint32_t)__cvta_generic_to_shared(mblk + lane);
                for (uint32_t w = 0; w < Wi; ++w)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dsts + w * 128u), "l"(src + w * 32) : "memory");
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
            // candidate of bit 0 of every mask word of this cell's rows
            uint16_t *wq = (uint32_t)wbcap > kWqCap ? wq_dyn : wqtab[warp];
            uint32_t W = 0;
            {
                const int zlo = DIM == 3 ? -1 : 0, zhi = DIM == 3 ? 1 : 0;
                for (int dz = zlo; dz <= zhi; ++dz) {
                    const int sz = sl[2] + dz;
                    if (DIM == 3 && (sz < 0 || sz >= tt.ext[2])) continue;
                    for (int dy = -1; dy <= 1; ++dy) {
                        const int sy = sl[1] + dy;
                        if (sy < 0 || sy >= tt.ext[1]) continue;
                        const int rowbase = tt.ext[0] * (sy + tt.ext[1] * sz);
                        const int xa = max(sl[0] - 1, 0), xb = min(sl[0] + 1, tt.ext[0] - 1);
                        const uint32_t q0 = tt.h_off[rowbase + xa], q1 = tt.h_off[rowbase + xb + 1];
                        const uint32_t nb = (q1 - q0 + 31u) >> 5;
                        for (uint32_t bb = lane; bb < nb; bb += 32)
                            if (W + bb < wqcap) wq[W + bb] = (uint16_t)(min(q0 + 32u * bb + 32u, q1) - 1u);
                        W += nb;
                    }
                }
            }
            uint32_t n = 0;
            if (W <= wqcap && W <= (uint32_t)wbcap) {
                // the item's mask block into shared memory (coalesced), then every lane walks its own column at its
                // own pace (no per-word reconvergence): ~hits + words iterations instead of sum over words of the
                // largest popcount of the warp
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                __syncwarp();
                // one flat loop, byte addresses kept in registers: an iteration either fetches the lane's next mask
                // word or emits one hit
                uint32_t maddr = (uint32_t)__cvta_generic_to_shared(mblk + (active ? lane : 0));
                uint32_t waddr = (uint32_t)__cvta_generic_to_shared(wq);
                const uint32_t mend = maddr + W * 128u;
                uint32_t m = 0, qtop = 0;
                if (staged) {
                    uint32_t daddr = (uint32_t)__cvta_generic_to_shared(dst_s);
                    // One predicated instruction block per iteration (no divergent branch: with branches the lanes
                    // split into independently scheduled fragments and the instruction count triples): a lane whose
                    // word is empty fetches its next word, any other lane emits its highest set bit (ascending
                    // candidates = descending bits).  The warp vote ends the loop for all lanes together.
                    for (;;) {
                        asm volatile(
                            "{\n"
                            ".reg .pred pe, pf;\n"
                            ".reg .u32 hb, v, bit;\n"
                            "setp.eq.u32 pe, %0, 0;\n"
                            "setp.ne.and.u32 pf, %2, %5, pe;\n"
                            "@!pe bfind.u32 hb, %0;\n"
                            "@!pe sub.u32 v, %1, hb;\n"
                            "@!pe st.shared.u16 [%3], v;\n"
                            "@!pe add.u32 %3, %3, 2;\n"
                            "@!pe shl.b32 bit, 1, hb;\n"
                            "@!pe xor.b32 %0, %0, bit;\n"
                            "@pf ld.shared.u32 %0, [%2];\n"
                            "@pf ld.shared.u16 %1, [%4];\n"
                            "@pf add.u32 %2, %2, 128;\n"
                            "@pf add.u32 %4, %4, 2;\n"
                            "}\n"
                            : "+r"(m), "+r"(qtop), "+r"(maddr), "+r"(daddr), "+r"(waddr)
                            : "r"(mend)
                            : "memory");
                        if (__all_sync(0xffffffffu, m == 0 && maddr == mend)) break;
                    }
                } else {
                    for (;;) {
                        if (m == 0) {
                            if (maddr == mend) break;
                            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(m) : "r"(maddr));
                            asm volatile("ld.shared.u16 %0, [%1];" : "=r"(qtop) : "r"(waddr));
                            maddr += 128u;
                            waddr += 2u;
                        } else {
                            const uint32_t hb = 31u - (uint32_t)__clz(m);
                            m ^= 1u << hb;
                            dst_g[n++] = (uint16_t)(qtop - hb);
                        }
                    }
                }
            } else {
                __syncwarp();
                const int zlo = DIM == 3 ? -1 : 0, zhi = DIM == 3 ? 1 : 0;
                for (int dz = zlo; dz <= zhi; ++dz) {
                    const int sz = sl[2] + dz;
                    if (DIM == 3 && (sz < 0 || sz >= tt.ext[2])) continue;
                    for (int dy = -1; dy <= 1; ++dy) {
                        const int sy = sl[1] + dy;
                        if (sy < 0 || sy >= tt.ext[1]) continue;
                        const int rowbase = tt.ext[0] * (sy + tt.ext[1] * sz);
                        const int xa = max(sl[0] - 1, 0), xb = min(sl[0] + 1, tt.ext[0] - 1);
                        const uint32_t q0 = tt.h_off[rowbase + xa], q1 = tt.h_off[rowbase + xb + 1];
                        for (uint32_t q = q0; q < q1; q += 32, mp += 32) {
                            const uint32_t qtop = min(q + 32u, q1) - 1u;       // candidate of bit 0
                            uint32_t m = *mp;
                            while (m) {
                                const int hb = 31 - __clz(m);
                                m ^= 1u << hb;
                                const uint16_t v = (uint16_t)(qtop - (uint32_t)hb);
                                if (staged) dst_s[n] = v; else dst_g[n] = v;
                                ++n;
                            }
                        }
                    }
                }
            }
            if (staged) {
                __syncwarp();
                uint16_t *out = col16 + seg0;
                for (uint32_t k = lane; k < total; k += 32) out[k] = wbuf[k];
                __syncwarp();
            }
        }
    }
}

// ---------------------------------------------------------------------------------------- tile statistics
// largest halo population and largest row count over all tiles of a candidate decomposition (one thread per tile)
template <int DIM>
__global__ void k_tile_stats(TileGeom tg, const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
                             uint32_t *__restrict__ out /* [2]: Mmax, Tmax */, uint32_t *__restrict__ occ_out,
                             uint32_t *__restrict__ half_out /* or NULL: largest halo of HALF a tile (k_vjp_tile) */)
{
    const int tile = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t M = 0, T = 0, occ = 0, Mh = 0;
    uint32_t slab[4] = {0u, 0u, 0u, 0u};                    // halo particles per z-layer of cells (B <= 2 in 3D)
    if (tile < tg.ntiles) {
        int b = tile, bc[3] = {0, 0, 0};
        bc[0] = b % tg.nb[0];
        b /= tg.nb[0];
        bc[1] = b % tg.nb[1];
        bc[2] = b / tg.nb[1];
        int lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, t0[3] = {0, 0, 0}, t1[3] = {0, 0, 0};   // inclusive ranges (unwrapped)
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
            const int c0 = bc[k] * tg.B, tn = min(tg.B, tg.ncell[k] - c0);
            t0[k] = c0;
            t1[k] = c0 + tn - 1;
            lo[k] = tg.periodic[k] ? c0 - 1 : max(c0 - 1, 0);
            hi[k] = tg.periodic[k] ? c0 + tn : min(c0 + tn, tg.ncell[k] - 1);
        }
        for (int cz = lo[2]; cz <= hi[2]; ++cz)
            for (int cy = lo[1]; cy <= hi[1]; ++cy)
                for (int cx = lo[0]; cx <= hi[0]; ++cx) {
                    int c[3] = {cx, cy, cz};
                    bool tgt = true;
                    int64_t lin = 0;
#pragma unroll
                    for (int k = DIM - 1; k >= 0; --k) {
                        tgt = tgt && c[k] >= t0[k] && c[k] <= t1[k];
                        int w = c[k];
                        if (tg.periodic[k]) w = w < 0 ? w + tg.ncell[k] : (w >= tg.ncell[k] ? w - tg.ncell[k] : w);
                        lin = lin * tg.ncell[k] + w;
                    }
                    const uint32_t cc = cell_end[lin] - cell_start[lin];
                    M += cc;
                    if (DIM == 3 && cz - lo[2] < 4) slab[cz - lo[2]] += cc;
                    if (tgt) T += cc;
                    occ = max(occ, cc);
                }
        // a tile of two cell layers in z can be worked on as two halves, each with the three layers around its own
        if (DIM == 3 && half_out) {
            if (t1[2] - t0[2] != 1) Mh = M;
            else
                for (int s = 0; s < 2; ++s) {
                    uint32_t m = 0;
                    for (int cz = max(t0[2] + s - 1, lo[2]); cz <= min(t0[2] + s + 1, hi[2]); ++cz) m += slab[cz - lo[2]];
                    Mh = max(Mh, m);
                }
        }
    }
    M = __reduce_max_sync(0xffffffffu, M);
    T = __reduce_max_sync(0xffffffffu, T);
    Mh = __reduce_max_sync(0xffffffffu, Mh);
    occ = __reduce_max_sync(0xffffffffu, occ);
    if ((threadIdx.x & 31) == 0) {
        atomicMax(&out[0], M);
        atomicMax(&out[1], T);
        atomicMax(occ_out, occ);                     // largest cell occupancy
        if (half_out) atomicMax(half_out, Mh);
    }
}

// tables of every tile, once per build: the tile kernels then load theirs instead of deriving it (sph_tiles.cuh)
template <int DIM>
__global__ void __launch_bounds__(64)
k_tile_tables(TileGeom tg, const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end, TileTab *__restrict__ out)
{
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);          // tg.tabs is NULL here
    const uint32_t *src = reinterpret_cast<const uint32_t *>(&tt);
    uint32_t *dst = reinterpret_cast<uint32_t *>(out + blockIdx.x);
    for (int i = threadIdx.x; i < (int)(sizeof(TileTab) / 4); i += blockDim.x) dst[i] = src[i];
}

// ---------------------------------------------------------------------------------------- col16 -> sorted ids
// (export and the generic pair kernels only) one CTA per tile; rows of a tile are contiguous
template <int DIM>
__global__ void __launch_bounds__(256)
k_expand_col16(TileGeom tg, const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
               const long long *__restrict__ row_ptr, const uint16_t *__restrict__ col16, int32_t *__restrict__ col,
               uint32_t mapcap)
{
    extern __shared__ uint32_t qmap[];                    // [mapcap] halo-linear index -> sorted index, when the halo fits
    __shared__ TileTab tt;
    tile_setup<DIM>(tg, blockIdx.x, cell_start, cell_end, tt);
    if (tt.T == 0) return;
    const long long b = row_ptr[tt.row0], e = row_ptr[tt.row0 + tt.T];
    if (tt.M <= mapcap) {
        // one table look-up per entry instead of a binary search over the halo cells
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
        for (int hc = warp; hc < tt.nh; hc += nwarps) {
            const uint32_t o0 = tt.h_off[hc], cnt = tt.h_off[hc + 1] - o0, gs = tt.h_start[hc];
            for (uint32_t l = lane; l < cnt; l += 32) qmap[o0 + l] = gs + l;
        }
        __syncthreads();
        for (long long p = b + threadIdx.x; p < e; p += blockDim.x) col[p] = (int32_t)qmap[col16[p]];
    } else {
        for (long long p = b + threadIdx.x; p < e; p += blockDim.x) col[p] = (int32_t)tile_q_to_sorted(tt, col16[p]);
    }
}

} // namespace

// ==========================================================================================
// host side
// ==========================================================================================
static TileGeom make_tile_geom(const GridGeom &gg, int B)
{
    TileGeom tg;
    memset(&tg, 0, sizeof(tg));
    tg.dim = gg.dim;
    tg.B = B;
    tg.ntiles = 1;
    for (int k = 0; k < 3; ++k) {
        tg.nb[k] = 1;
        tg.ncell[k] = gg.ncell[k];
        tg.periodic[k] = gg.periodic[k];
        tg.L[k] = gg.L[k];
        if (k < gg.dim) tg.nb[k] = (gg.ncell[k] + B - 1) / B;
        tg.ntiles *= tg.nb[k];
    }
    return tg;
}

static bool tile_geom_ok(const GridGeom &gg, int B)
{
    int halo = 1, tgt = 1;
    for (int k = 0; k < gg.dim; ++k) {
        if (gg.periodic[k] && gg.ncell[k] < B + 2) return false;   // the halo would wrap onto itself
        halo *= B + 2;
        tgt *= B;
    }
    return halo <= kTileMaxHalo && tgt <= kTileMaxTgt;
}

// candidate tile edges of a dimension, best first
int sph_tile_candidates(const sph_ctx *ctx, int out[3])
{
    const GridGeom &gg = ctx->geom;
    int n = 0;
    const int pref3[2] = {2, 1}, pref2[3] = {4, 2, 1};
    const int *pref = gg.dim == 3 ? pref3 : pref2;
    const int np = gg.dim == 3 ? 2 : 3;
    for (int i = 0; i < np; ++i) {
        if (ctx->opt_tile_edge && pref[i] != ctx->opt_tile_edge) continue;
        if (tile_geom_ok(gg, pref[i])) out[n++] = pref[i];
    }
    return n;
}

// enqueue the statistics of every candidate decomposition into stats[4 + 2k], stats[5 + 2k]
int sph_tile_stats_launch(sph_ctx *ctx, const int *cand, int ncand, cudaStream_t st)
{
    uint32_t *stats = ctx->stats.as<uint32_t>();
    SPH_CUDA_TRY(cudaMemsetAsync(stats + 4, 0, 7 * sizeof(uint32_t), st));
    SPH_CUDA_TRY(cudaMemsetAsync(stats + kTileHalfSlot, 0, sizeof(uint32_t), st));
    for (int k = 0; k < ncand; ++k) {
        const TileGeom tg = make_tile_geom(ctx->geom, cand[k]);
        KScope ks(ctx, SPH_K_COUNT, 1, st);
        const unsigned nb = (unsigned)((tg.ntiles + 127) / 128);
        if (tg.dim == 3)
            k_tile_stats<3><<<nb, 128, 0, st>>>(tg, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), stats + 4 + 2 * k, stats + 10,
                                                cand[k] == 2 ? stats + kTileHalfSlot : nullptr);
        else k_tile_stats<2><<<nb, 128, 0, st>>>(tg, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), stats + 4 + 2 * k, stats + 10, nullptr);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

// shared-memory budget of the pair kernels decides which halo sizes the tile layout accepts
size_t sph_tile_state_bytes(int dim) { return dim == 3 ? 56 : 48; }   // VJP: state + cotangents per halo particle
static const size_t kTileSmemBudget = 200 * 1024;

// the tile SEARCH only stages positions (16 B per halo particle): it fits far larger halos than the pair kernels.
// Its lists are then translated to sorted ids for the generic pair kernels (BASELINE config 4: 134 particles per cell).
bool sph_tile_search_fits(uint32_t Mmax)
{
    return Mmax > 0 && Mmax <= 65535u && (size_t)(Mmax + 8) * 16 + 8 * 2 * 4096 <= kTileSmemBudget;
}

bool sph_tile_fits(int dim, uint32_t Mmax)
{
    return Mmax > 0 && Mmax <= 65535u && (size_t)(Mmax + 8) * sph_tile_state_bytes(dim) + (size_t)(Mmax + 8) * 4 <= kTileSmemBudget;
}

// count / scan / fill of the tile-local lists with tile edge B.  Synchronises `st` once (nnz readback).
int sph_neighbors_tile_run(sph_ctx *ctx, const SearchPar &sp, int B, uint32_t Mmax, uint32_t Tmax, uint32_t occmax,
                           cudaStream_t st, int64_t *nnz_out)
{
    const int64_t n = ctx->n;
    const GridGeom &gg = ctx->geom;
    TileGeom tg = make_tile_geom(gg, B);
    if (ctx->opt_tile_tables) {
        SPH_TRY(ctx->tile_tabs.reserve((size_t)tg.ntiles * sizeof(TileTab)));
        KScope ks(ctx, SPH_K_COUNT, 1, st);
        if (gg.dim == 3)
            k_tile_tables<3><<<(unsigned)tg.ntiles, 64, 0, st>>>(tg, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), ctx->tile_tabs.as<TileTab>());
        else
            k_tile_tables<2><<<(unsigned)tg.ntiles, 64, 0, st>>>(tg, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), ctx->tile_tabs.as<TileTab>());
        tg.tabs = ctx->tile_tabs.p;
    }
    if (ctx->opt_build_fused && ctx->f_ncmax) {
        // the one-kernel build (sph_neighbors_fused.cu); 1 = a tile does not fit its shared-memory carve-up
        const int rc = sph_neighbors_fused_run(ctx, sp, tg, Mmax, Tmax, ctx->f_ncmax, ctx->f_pairs, st, nnz_out);
        if (rc != 1) return rc;
    }
    const bool varh = ctx->hmin != ctx->hmax;
    const int mcap = (int)((Mmax + 7u) & ~7u);
    SPH_TRY(ctx->cnt.reserve((size_t)n * 4));
    SPH_TRY(ctx->row_ptr.reserve((size_t)(n + 1) * 8));
    const float4 *pos = ctx->pos_s.as<float4>();
    const uint32_t *cs = ctx->cell_start.as<uint32_t>(), *ce = ctx->cell_end.as<uint32_t>();
    // hit masks of the count pass (so that the fill repeats no distance test): upper bound of the mask words from
    // the largest cell occupancy -- no extra readback.  Beyond 24 GB the fill recomputes the tests instead.
    uint32_t *maskbuf = nullptr;
    long long *mask_base = nullptr;
    {
        int nr = gg.dim == 3 ? 9 : 3;
        const double wmax = (double)nr * (double)((3u * occmax + 31u) / 32u);
        const double bound = ((double)n + 32.0 * (double)ctx->ncells_total) * wmax;
        if (ctx->opt_fill_masks && bound * 4.0 <= 24.0e9) {
            SPH_TRY(ctx->maskbuf.reserve((size_t)bound * 4 + 256));
            SPH_TRY(ctx->tile_words.reserve((size_t)tg.ntiles * 4));
            SPH_TRY(ctx->tile_mask_base.reserve((size_t)(tg.ntiles + 1) * 8));
            maskbuf = ctx->maskbuf.as<uint32_t>();
            mask_base = ctx->tile_mask_base.as<long long>();
            KScope ks(ctx, SPH_K_COUNT, 4, st);
            uint32_t *wmax_dev = ctx->stats.as<uint32_t>() + 11;       // largest number of mask words of a row
            SPH_CUDA_TRY(cudaMemsetAsync(wmax_dev, 0, 4, st));
            if (gg.dim == 3) k_tile_words<3><<<(unsigned)tg.ntiles, 64, 0, st>>>(tg, cs, ce, ctx->tile_words.as<uint32_t>(), wmax_dev);
            else k_tile_words<2><<<(unsigned)tg.ntiles, 64, 0, st>>>(tg, cs, ce, ctx->tile_words.as<uint32_t>(), wmax_dev);
            SPH_TRY(sph_scan_u32(ctx, ctx->tile_words.as<uint32_t>(), mask_base, true, tg.ntiles, st));
        }
    }
#define SPH_NBT_LAUNCH(DIM, FILL, VARH, SMEM, WCAP, CNT, RP, COL)                                                      \
    do {                                                                                                               \
        SPH_CUDA_TRY(cudaFuncSetAttribute(k_nb_tile<DIM, FILL, VARH>, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                                          (int)(SMEM)));                                                               \
        k_nb_tile<DIM, FILL, VARH><<<(unsigned)tg.ntiles, kNbWarps * 32, (SMEM), st>>>(                                \
            tg, gg, sp, mcap, (WCAP), pos, cs, ce, CNT, RP, COL, (FILL) ? nullptr : maskbuf, mask_base);               \
    } while (0)
#define SPH_NBT_DISPATCH(FILL, SMEM, WCAP, CNT, RP, COL)                                                               \
    do {                                                                                                               \
        if (gg.dim == 3) { if (varh) SPH_NBT_LAUNCH(3, FILL, true, SMEM, WCAP, CNT, RP, COL);                          \
                           else SPH_NBT_LAUNCH(3, FILL, false, SMEM, WCAP, CNT, RP, COL); }                            \
        else { if (varh) SPH_NBT_LAUNCH(2, FILL, true, SMEM, WCAP, CNT, RP, COL);                                      \
               else SPH_NBT_LAUNCH(2, FILL, false, SMEM, WCAP, CNT, RP, COL); }                                        \
    } while (0)
    {
        KScope ks(ctx, SPH_K_COUNT, 1, st);
        const size_t smem = (size_t)mcap * sizeof(float4);
        SPH_NBT_DISPATCH(false, smem, 0, ctx->cnt.as<uint32_t>(), nullptr, nullptr);
    }
    {
        KScope ks(ctx, SPH_K_SCAN, 3, st);
        SPH_TRY(sph_scan_u32(ctx, ctx->cnt.as<uint32_t>(), ctx->row_ptr.p, true, n, st));
    }
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->h_pinned + 4, ctx->row_ptr.as<long long>() + n, 8, cudaMemcpyDeviceToHost, st));
    if (maskbuf) SPH_CUDA_TRY(cudaMemcpyAsync(ctx->h_pinned + 5, ctx->stats.as<uint32_t>() + 11, 4, cudaMemcpyDeviceToHost, st));
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    const int64_t nnz = ctx->h_pinned[4];
    uint32_t wmax_rows = 0;
    if (maskbuf) memcpy(&wmax_rows, ctx->h_pinned + 5, 4);
    SPH_TRY(ctx->col16.reserve((size_t)(nnz > 0 ? nnz : 1) * 2 + 64));
    {
        // per-warp staging capacity: 32 rows of the mean length with head room; the halo positions come first
        const double mean = (double)nnz / (double)n;
        int wcap = (int)(32.0 * mean * 1.35) + 64;
        wcap = (wcap + 63) & ~63;
        if (wcap < 512) wcap = 512;
        const size_t pos_bytes = (size_t)mcap * sizeof(float4);
        const size_t budget = pos_bytes > 48 * 1024 ? 200 * 1024 : 100 * 1024;   // two CTAs per SM when the halo is small
        if (pos_bytes + (size_t)kNbWarps * wcap * 2 > budget) {
            const size_t room = pos_bytes < budget ? budget - pos_bytes : 0;
            int w2 = (int)(room / (kNbWarps * 2)) & ~63;
            if (w2 < 512) w2 = 512;
            if (w2 < wcap) wcap = w2;
        }
        KScope ks(ctx, SPH_K_FILL, 1, st);
        if (maskbuf) {
            int wc = (int)(32.0 * mean * 1.2) + 64;
            wc = (wc + 63) & ~63;
            if (wc < 512) wc = 512;
            if (wc > 12288) wc = 12288;
            int wb = (int)wmax_rows;                            // most mask words any row has (k_tile_words)
            if (wb < 1) wb = 1;
            // rows with up to 64 mask words (the usual case): 4 warps per CTA, static word table.  Dense cells (config 4:
            // ~190 words per row): the mask block of an item is up to 28 KB, so 2 warps per CTA keep three CTAs per SM;
            // rows beyond 224 words take the word-synchronous expansion
            if (wb > 224) wb = 224;
            const int ew = wb > 64 ? 2 : 4;                                         // warps per CTA
            const size_t smem = (size_t)ew * ((size_t)wc * 2 + (size_t)wb * 128 + ((uint32_t)wb > kWqCap ? (size_t)wb * 2 : 0)) + 16;
            if (gg.dim == 3) {
                SPH_CUDA_TRY(cudaFuncSetAttribute(k_nb_expand<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                k_nb_expand<3><<<(unsigned)tg.ntiles, ew * 32, smem, st>>>(tg, wc, wb, cs, ce, ctx->row_ptr.as<long long>(),
                                                                               ctx->col16.as<uint16_t>(), maskbuf, mask_base);
            } else {
                SPH_CUDA_TRY(cudaFuncSetAttribute(k_nb_expand<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                k_nb_expand<2><<<(unsigned)tg.ntiles, ew * 32, smem, st>>>(tg, wc, wb, cs, ce, ctx->row_ptr.as<long long>(),
                                                                               ctx->col16.as<uint16_t>(), maskbuf, mask_base);
            }
        } else {
        const size_t smem = pos_bytes + (size_t)kNbWarps * wcap * 2;
        SPH_NBT_DISPATCH(true, smem, wcap, nullptr, ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>());
        }
    }
#undef SPH_NBT_DISPATCH
#undef SPH_NBT_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    ctx->tg = tg;
    ctx->tile_mode = true;
    ctx->tile_Mmax = Mmax;
    ctx->tile_Tmax = Tmax;
    ctx->col_valid = false;
    ctx->nnz = nnz;
    ctx->n_lists = n;
    if (nnz_out) *nnz_out = nnz;
    return SPH_OK;
}

// materialise the 32-bit sorted-id lists from the tile-local ones (export; generic pair kernels)
int sph_tile_expand_col(sph_ctx *ctx, cudaStream_t st)
{
    if (!ctx->tile_mode || ctx->col_valid) return SPH_OK;
    SPH_TRY(ctx->col.reserve((size_t)(ctx->nnz > 0 ? ctx->nnz : 1) * 4));
    KScope ks(ctx, SPH_K_EXPORT, 1, st);
    const TileGeom &tg = ctx->tg;
    const uint32_t mapcap = ctx->tile_Mmax <= 11000u ? ctx->tile_Mmax : 0u;     // 44 KB of dynamic shared memory at most
    const size_t smem = (size_t)mapcap * 4;
    if (tg.dim == 3)
        k_expand_col16<3><<<(unsigned)tg.ntiles, 256, smem, st>>>(tg, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),
                                                                 ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->col.as<int32_t>(), mapcap);
    else
        k_expand_col16<2><<<(unsigned)tg.ntiles, 256, smem, st>>>(tg, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(),
                                                                 ctx->row_ptr.as<long long>(), ctx->col16.as<uint16_t>(), ctx->col.as<int32_t>(), mapcap);
    SPH_CUDA_TRY(cudaGetLastError());
    ctx->col_valid = true;
    return SPH_OK;
}
