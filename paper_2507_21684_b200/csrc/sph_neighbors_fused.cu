// sph_neighbors_fused.cu -- steps N5 + N6 + N7 of SURVEY.md 8(a) (count, offsets, fill of the tile-local compact lists;
// PAPER.md:556-558 App. B steps 1-3, PAPER.md:163 pair list, PAPER.md:167 radius max{h_i,h_j}) as ONE tile-resident
// kernel.  The two-kernel build of sph_neighbors_tile.cu wrote every hit mask to HBM so that the fill could read it
// back (6.2x / 1.65x the algorithmic DRAM bytes, profiles/r01_d); here a tile's masks never leave shared memory:
//
//   phase 1  tests.  A lane owns 4 candidates of one target cell (their positions stay in registers); the rows of the
//            cell stream past as PAIRS -- {x_a,x_b,y_a,y_b},{z_a,z_b,h_a,h_b}, two broadcast loads serving 8 tests per
//            lane -- and the distance test of both rows is one chain of packed FP32 instructions (FADD2/FFMA2, sm_100a):
//            diff = fma(dz,dz, fma(dy,dy, fma(dx,dx, -Hs^2))), the same IEEE operations in the same order as the
//            scalar test, so the fp32 verdicts and the "too close to call" band (reading R3: resolved by the binary64
//            predicate) are unchanged.  The verdict is the sign bit, funnel-shifted into a per-candidate mask over rows;
//            a 32x32 bit transpose across the warp turns it into per-row masks over candidates in shared memory.
//   phase 2  per-row counts (popcounts of the masks), CTA scan, and the tile's base offset from a decoupled look-back
//            over the tiles in Morton order (the order of their rows in the sorted arrays); status and value travel in
//            one 64-bit word, so no fence is needed.  row_ptr and cnt are written here.
//   phase 3  expansion of the masks into uint16 halo indices in a shared-memory image of the tile's contiguous col16
//            segment (two lanes per row, one flat predicated loop: an iteration fetches the lane's next mask word or
//            emits one hit), flushed with 16-byte stores.
// Deterministic: fixed candidate order, no float atomics; the only atomics are the ticket counter and integer flags.
#include "sph_internal.cuh"
#include "sph_tiles.cuh"
#include "sph_search.cuh"

#include <math.h>

#include <algorithm>
#include <vector>

namespace {

constexpr int kFWmax = 16;             // warps per CTA (launch bound)
constexpr int kRowLanes = 4;           // lanes that share a row in the expansion (phase 3)
constexpr int kCPL = 4;                // candidates per lane in the test loop
constexpr int kCandBlock = 32 * kCPL;  // candidates per work unit
constexpr uint32_t kQNone = 0xffffu;   // padding entry of a candidate map

struct FusedSizes {
    int mcap;            // halo particles (multiple of 8)
    int tcap;            // rows of a tile
    int ncap;            // candidates of one target cell, multiple of kCandBlock
    int wcap;            // mask words of a row = ceil(most candidates of a cell / 32) <= ncap / 32
    int pcap;            // row pairs of a tile
    int scap;            // entries of the staging image (multiple of 8)
    int nt_max;          // target cells of a tile
    long long col_cap;   // capacity of col16 in entries
};

constexpr unsigned long long kFlagAgg = 1ull << 62, kFlagPre = 2ull << 62, kValMask = (1ull << 62) - 1ull;

__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Decoupled look-back (single-pass prefix over the tiles in ticket order).  Called by all 32 lanes of warp 0.  Returns the
// exclusive prefix of `tot`.  A tile only waits on lower tickets, and tickets are handed out in the order the CTAs start.
__device__ __forceinline__ long long tile_lookback(unsigned long long *tstate, uint32_t ticket, uint32_t tot)
{
    const int lane = threadIdx.x & 31;
    if (ticket == 0) {
        if (lane == 0) st_volatile_u64(tstate, kFlagPre | (unsigned long long)tot);
        return 0;
    }
    if (lane == 0) st_volatile_u64(tstate + ticket, kFlagAgg | (unsigned long long)tot);
    unsigned long long excl = 0;
    long long pos = (long long)ticket - 1;
    for (;;) {
        const long long idx = pos - lane;
        unsigned long long s;
        for (;;) {
            s = idx >= 0 ? ld_volatile_u64(tstate + idx) : kFlagPre;
            if (!__any_sync(0xffffffffu, (s >> 62) == 0ull)) break;
            __nanosleep(100);
        }
        const uint32_t pre = __ballot_sync(0xffffffffu, (s >> 62) == 2ull);
        unsigned long long v = s & kValMask;
        if (pre) {
            const int first = __ffs(pre) - 1;            // closest predecessor that already knows its prefix
            if (lane > first) v = 0;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        excl += v;
        if (pre) break;
        pos -= 32;
    }
    if (lane == 0) st_volatile_u64(tstate + ticket, kFlagPre | (excl + (unsigned long long)tot));
    return (long long)excl;
}

// 32x32 bit transpose across the lanes of a warp (five butterfly stages).  With x_l the word of lane l, the result y of
// lane b has   bit l of y_b  =  bit (31 - b) of x_{31 - l}   (the transpose about the anti-diagonal).
__device__ __forceinline__ uint32_t warp_transpose32(uint32_t x)
{
    const int lane = threadIdx.x & 31;
    uint32_t m = 0x0000ffffu;
#pragma unroll
    for (int j = 16; j > 0; j >>= 1) {
        const uint32_t p = __shfl_xor_sync(0xffffffffu, x, j);
        if ((lane & j) == 0) {
            const uint32_t t = (x ^ (p >> j)) & m;
            x ^= t;
        } else {
            const uint32_t t = (p ^ (x >> j)) & m;
            x ^= t << j;
        }
        m ^= m << (j >> 1);
    }
    return x;
}

// Tile-relative coordinate (x + sh) - o of a halo particle: sh = 0 or -+L moves a cell across a periodic face, o is the
// tile's corner.  x + sh is formed exactly as hi + lo (TwoSum), hi - o is exact (both lie within a few cells of each
// other), so the result carries one rounding at the magnitude of the TILE, not of the box: differences of two such
// coordinates are good to ~2^-24 of a few cell edges on every tile, seam or not, and one tolerance band serves all.
__device__ __forceinline__ float rel_coord(float x, float sh, float o)
{
    const float hi = __fadd_rn(x, sh);
    const float bb = __fsub_rn(hi, x);
    const float lo = __fadd_rn(__fsub_rn(x, __fsub_rn(hi, bb)), __fsub_rn(sh, bb));
    return __fadd_rn(__fsub_rn(hi, o), lo);
}

// halo slot coordinates of halo cell hc
__device__ __forceinline__ void halo_slot(const TileTab &tt, int hc, int sl[3])
{
    sl[0] = hc % tt.ext[0];
    sl[1] = (hc / tt.ext[0]) % tt.ext[1];
    sl[2] = hc / (tt.ext[0] * tt.ext[1]);
}

// Visits the 3^(d-1) candidate runs [q0, q1) (halo-linear indices) of the target cell at halo slot sl, in (z, y) order.
template <int DIM, class F>
__device__ __forceinline__ void for_each_run(const TileTab &tt, const int sl[3], F f)
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
            f(tt.h_off[rowbase + xa], tt.h_off[rowbase + xb + 1]);
        }
    }
}

struct FusedSmem {
    float4 *cand;        // [mcap]   halo positions, shifted across periodic seams
    float4 *rp2;         // [2 pcap] row pairs: {x_a,x_b,y_a,y_b}, {z_a,z_b,h_a,h_b}
    uint16_t *stage;     // [scap + 8] image of a col16 segment; OVERLAYS cand / rp2 (dead after phase 1)
    uint32_t *masks;     // [wcap][tcap]  hit masks, candidate c of word w at bit 31 - c
    uint16_t *cmap;      // [nt][ncap]    candidate g of target cell tc -> halo-linear index
    uint32_t *off;       // [tcap + 1]    counts, then exclusive offsets
    uint16_t *qcnt;      // [3 tcap]      hits before the 2nd, 3rd, 4th lane of a row (phase 3)
    uint8_t *qwrd;       // [3 tcap]      first mask word of the 2nd, 3rd, 4th lane of a row
    uint8_t *rowcell;    // [tcap]        target cell of a row
    __device__ FusedSmem(unsigned char *base, const FusedSizes &fs)
    {
        size_t o = 0;
        cand = reinterpret_cast<float4 *>(base);
        rp2 = cand + fs.mcap;
        stage = reinterpret_cast<uint16_t *>(base);
        size_t r0 = (size_t)fs.mcap * 16 + (size_t)fs.pcap * 32, r1 = (size_t)(fs.scap + 8) * 2;
        o = ((r0 > r1 ? r0 : r1) + 15) & ~(size_t)15;
        masks = reinterpret_cast<uint32_t *>(base + o); o += (size_t)fs.wcap * fs.tcap * 4;
        cmap = reinterpret_cast<uint16_t *>(base + o); o += (size_t)fs.nt_max * fs.ncap * 2;
        o = (o + 3) & ~(size_t)3;
        off = reinterpret_cast<uint32_t *>(base + o); o += (size_t)(fs.tcap + 1) * 4;
        qcnt = reinterpret_cast<uint16_t *>(base + o); o += (size_t)fs.tcap * 6;
        rowcell = reinterpret_cast<uint8_t *>(base + o); o += (size_t)fs.tcap;
        qwrd = reinterpret_cast<uint8_t *>(base + o);
    }
};
// bytes behind the overlay region, and the whole carve-up (must mirror FusedSmem)
size_t fused_fixed_bytes(const FusedSizes &fs)
{
    size_t o = (size_t)fs.wcap * fs.tcap * 4 + (size_t)fs.nt_max * fs.ncap * 2;
    o = (o + 3) & ~(size_t)3;
    o += (size_t)(fs.tcap + 1) * 4 + (size_t)fs.tcap * 6 + (size_t)fs.tcap * 4 + 16;
    return o;
}
size_t fused_smem_bytes(const FusedSizes &fs)
{
    const size_t r0 = (size_t)fs.mcap * 16 + (size_t)fs.pcap * 32, r1 = (size_t)(fs.scap + 8) * 2;
    return (((r0 > r1 ? r0 : r1) + 15) & ~(size_t)15) + fused_fixed_bytes(fs);
}

// ---------------------------------------------------------------------------------------------------- the kernel
// ctl[0] = ticket counter, ctl[1] = overflow flag (col16 too small: lists not written, counts still exact)
template <int DIM, bool VARH>
__global__ void __launch_bounds__(kFWmax * 32, 2)
k_nb_fused(TileGeom tg, GridGeom gg, SearchPar sp, FusedSizes fs, long long n, const float4 *__restrict__ pos_s,
           const uint32_t *__restrict__ cell_start, const uint32_t *__restrict__ cell_end,
           const uint32_t *__restrict__ tile_order, uint32_t *__restrict__ ctl, unsigned long long *__restrict__ tstate,
           uint32_t *__restrict__ cnt_out, long long *__restrict__ row_ptr, uint16_t *__restrict__ col16)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const FusedSmem sm(smem_raw, fs);
    __shared__ TileTab tt;
    // per target cell: candidates, first row pair, first row (relative to the tile's first SORTED row: the rows of a tile
    // follow the Morton order of its cells, not the raster order of the target-cell table)
    __shared__ uint32_t c_nc[kTileMaxTgt], c_pb[kTileMaxTgt + 1], c_rb[kTileMaxTgt], c_ub[kTileMaxTgt + 1];
    __shared__ uint32_t s_ticket, s_tot, s_grp, s_hits;
    __shared__ volatile uint32_t s_ready;                    // set once the look-back has produced s_base
    __shared__ volatile uint32_t s_off_ready;                // set once off[] (the row offsets of the tile) is complete
    __shared__ long long s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, kFW = blockDim.x >> 5;
    if (threadIdx.x == 0) {
        s_ticket = atomicAdd(&ctl[0], 1u);
        s_grp = 0;
        s_ready = 0;
        s_off_ready = 0;
        s_hits = 0;
    }
    __syncthreads();
    const uint32_t ticket = s_ticket;
    tile_setup<DIM>(tg, (int)tile_order[ticket], cell_start, cell_end, tt);
    const uint32_t T = tt.T;
    if (T == 0) {                                            // an empty tile still takes part in the prefix
        if (warp == 0) (void)tile_lookback(tstate, ticket, 0u);
        return;
    }
    const bool seam = tt.seam != 0;
    const int tcap = fs.tcap, ncap = fs.ncap;

    // ---- stage the halo positions, relative to the tile's corner (shifted across periodic seams)
    float org[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < DIM; ++k) org[k] = (float)(gg.lo_d[k] + (double)(tt.hs[k] + tt.tlo[k]) * gg.edge[k]);
    for (int hc = warp; hc < tt.nh; hc += kFW) {
        const uint32_t o0 = tt.h_off[hc], o1 = tt.h_off[hc + 1];
        if (o1 == o0) continue;
        float sh[3];
        tile_cell_shift<DIM>(tg, tt, hc, sh);
        const uint32_t gs = tt.h_start[hc];
        for (uint32_t q = o0 + lane; q < o1; q += 32) {
            float4 pj = pos_s[gs + (q - o0)];
            pj.x = rel_coord(pj.x, sh[0], org[0]);
            pj.y = rel_coord(pj.y, sh[1], org[1]);
            if (DIM == 3) pj.z = rel_coord(pj.z, sh[2], org[2]);
            SPH_ASSERT(q < (uint32_t)fs.mcap);
            sm.cand[q] = pj;
        }
    }
    // ---- candidate maps: candidate g of target cell tc -> halo-linear index (its 3^(d-1) runs concatenated)
    for (int tc = warp; tc < tt.nt; tc += kFW) {
        int sl[3];
        halo_slot(tt, tt.t_cell[tc], sl);
        uint16_t *cm = sm.cmap + (size_t)tc * ncap;
        uint32_t g = 0;
        for_each_run<DIM>(tt, sl, [&](uint32_t q0, uint32_t q1) {
            SPH_ASSERT(g + (q1 - q0) <= (uint32_t)ncap && q1 <= (uint32_t)fs.mcap);
            for (uint32_t i = lane; i < q1 - q0; i += 32) cm[g + i] = (uint16_t)(q0 + i);
            g += q1 - q0;
        });
        const uint32_t gpad = (g + kCandBlock - 1) / kCandBlock * kCandBlock;
        SPH_ASSERT(gpad <= (uint32_t)ncap);
        for (uint32_t i = g + lane; i < gpad; i += 32) cm[i] = (uint16_t)kQNone;
        if (lane == 0) c_nc[tc] = g;
    }
    if (threadIdx.x == 0) {
        uint32_t pb = 0;
        for (int tc = 0; tc < tt.nt; ++tc) {
            c_pb[tc] = pb;
            pb += (tt.t_off[tc + 1] - tt.t_off[tc] + 1u) >> 1;
            c_rb[tc] = tt.h_start[tt.t_cell[tc]] - tt.row0;
        }
        c_pb[tt.nt] = pb;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        // work units of phase 1 per target cell: (chunks of up to 64 rows) x (blocks of 128 candidates)
        uint32_t ub = 0;
        for (int tc = 0; tc < tt.nt; ++tc) {
            c_ub[tc] = ub;
            const uint32_t nrow = tt.t_off[tc + 1] - tt.t_off[tc], Nc = c_nc[tc];
            ub += ((nrow + 63u) >> 6) * ((Nc + kCandBlock - 1) / kCandBlock);
        }
        c_ub[tt.nt] = ub;
    }
    // ---- row pairs (rows of one cell, two by two; an odd last row is paired with itself) and the row -> cell table
    for (uint32_t r = threadIdx.x; r < T; r += blockDim.x) {
        int tc = 0;
        while (tc + 1 < tt.nt && !(r - c_rb[tc] < tt.t_off[tc + 1] - tt.t_off[tc])) ++tc;      // unsigned: r in [c_rb, c_rb + nrow)
        const uint32_t local = r - c_rb[tc], nrow = tt.t_off[tc + 1] - tt.t_off[tc];
        const float4 p = sm.cand[tt.h_off[tt.t_cell[tc]] + local];          // target cells are never shifted
        float *pr = reinterpret_cast<float *>(sm.rp2 + 2 * (size_t)(c_pb[tc] + (local >> 1)));
        const int side = (int)(local & 1u);
        pr[0 + side] = p.x; pr[2 + side] = p.y; pr[4 + side] = p.z; pr[6 + side] = p.w;
        if (side == 0 && local + 1 == nrow) { pr[1] = p.x; pr[3] = p.y; pr[5] = p.z; pr[7] = p.w; }
        sm.rowcell[r] = (uint8_t)tc;
    }
    __syncthreads();

    // ---- phase 1: tests.  Work unit = (target cell, block of 128 candidates, chunk of 32 rows).
    {
        const float Hs2_u = sp.Hs_u * sp.Hs_u;
        // band of the fp32 verdict: sp.band covers the rounding of the FMA chain, as much again the rounding of the
        // tile-relative coordinates (at most 2 Hs x 2^-24 x 8 Hs = 2^-20 Hs^2)
        const float band = 2.0f * sp.band;
        const float tol_u = band * Hs2_u;
        const float2 nHs2_u = make_float2(-Hs2_u, -Hs2_u);
        // units are dealt round-robin; inside a cell the candidate block runs fastest, so the (smaller) units of a
        // cell's last row chunk spread over the warps like the full ones
        int tc = 0;
        uint32_t my_hits = 0;                               // hits of the lane's candidates: the tile's total is known after phase 1
        for (uint32_t unit = warp; unit < c_ub[tt.nt]; unit += kFW) {
                {
                    while (unit >= c_ub[tc + 1]) ++tc;
                    const uint32_t nrow = tt.t_off[tc + 1] - tt.t_off[tc], Nc = c_nc[tc];
                    const int hc_i = tt.t_cell[tc];
                    const uint16_t *cm = sm.cmap + (size_t)tc * ncap;
                    const uint32_t ncb = (Nc + kCandBlock - 1) / kCandBlock;
                    const uint32_t rc = (unit - c_ub[tc]) / ncb, cb = (unit - c_ub[tc]) - rc * ncb;
                    // the cell's rows in nrc balanced chunks of an even number (<= 64) of rows
                    const uint32_t nrc = (nrow + 63u) >> 6, rpc = (((nrow + nrc - 1u) / nrc) + 1u) & ~1u;
                    const uint32_t r_lo = rc * rpc, nr = min(rpc, nrow - r_lo);          // rows [r_lo, r_lo + nr) of the cell
                    const uint32_t nr1 = min(nr, 32u), nr2 = nr - nr1;                  // first / second mask word over rows
                    const uint32_t np1 = (nr1 + 1u) >> 1, np2 = (nr2 + 1u) >> 1;
                    const float4 *rp = sm.rp2 + 2 * (size_t)(c_pb[tc] + (r_lo >> 1));
                    float2 nx[kCPL], ny[kCPL], nz[kCPL];
                    float hj[kCPL], amin[kCPL];
                    uint32_t rb[kCPL], rb2[kCPL], qk[kCPL];
#pragma unroll
                    for (int k = 0; k < kCPL; ++k) {
                        SPH_ASSERT(cb * kCandBlock + k * 32 + lane < (uint32_t)ncap);
                        qk[k] = cm[cb * kCandBlock + k * 32 + lane];
                        SPH_ASSERT(qk[k] == kQNone || qk[k] < (uint32_t)fs.mcap);
                        float4 pj = make_float4(1.0e18f, 1.0e18f, DIM == 3 ? 1.0e18f : 0.f, 0.f);   // padding: never a hit
                        if (qk[k] != kQNone) pj = sm.cand[qk[k]];
                        nx[k] = make_float2(-pj.x, -pj.x);
                        ny[k] = make_float2(-pj.y, -pj.y);
                        nz[k] = make_float2(-pj.z, -pj.z);
                        hj[k] = pj.w;
                        amin[k] = 3.0e38f;
                        rb[k] = 0u;
                        rb2[k] = 0u;
                    }
                    // one pair of rows against the lane's four candidates; the verdicts are shifted into `bits`
                    auto test_pair = [&](uint32_t p, uint32_t (&bits)[kCPL]) {
                        const float4 A = rp[2 * p], Bz = rp[2 * p + 1];
                        const float2 xa = make_float2(A.x, A.y), ya = make_float2(A.z, A.w), za = make_float2(Bz.x, Bz.y);
#pragma unroll
                        for (int k = 0; k < kCPL; ++k) {
                            const float2 d0 = __fadd2_rn(xa, nx[k]), d1 = __fadd2_rn(ya, ny[k]);
                            float2 nH = nHs2_u, tl = make_float2(0.f, 0.f);
                            if (VARH) {
                                const float2 Hs = __fmul2_rn(make_float2(fmaxf(Bz.z, hj[k]), fmaxf(Bz.w, hj[k])),
                                                             make_float2(sp.scale, sp.scale));
                                nH = __fmul2_rn(Hs, make_float2(-Hs.x, -Hs.y));
                                tl = __fmul2_rn(make_float2(-nH.x, -nH.y), make_float2(band, band));
                            }
                            float2 acc = __ffma2_rn(d0, d0, nH);
                            acc = __ffma2_rn(d1, d1, acc);
                            if (DIM == 3) {
                                const float2 d2 = __fadd2_rn(za, nz[k]);
                                acc = __ffma2_rn(d2, d2, acc);
                            }
                            bits[k] = __funnelshift_l(__float_as_uint(acc.x), bits[k], 1);   // (bits << 1) | (diff < 0)
                            bits[k] = __funnelshift_l(__float_as_uint(acc.y), bits[k], 1);
                            amin[k] = fminf(amin[k], fminf(fabsf(acc.x) - tl.x, fabsf(acc.y) - tl.y));
                        }
                    };
#pragma unroll 2
                    for (uint32_t p = 0; p < np1; ++p) test_pair(p, rb);
                    for (uint32_t p = 0; p < np2; ++p) test_pair(16u + p, rb2);
                    // row slot i of the first word sits at bit 2 np1 - 1 - i of rb[k], of the second at 2 np2 - 1 - (i - 32)
                    // of rb2[k].  Too close to call (rare, except on exact lattices): a second pass over the rows marks
                    // the pairs inside the band, and the binary64 predicate of reading R3 decides those.
#pragma unroll
                    for (int k = 0; k < kCPL; ++k) {
                        const bool flagged = qk[k] != kQNone && amin[k] <= (VARH ? 0.f : tol_u);
                        if (!__any_sync(0xffffffffu, flagged)) continue;
                        uint32_t nb1 = 0u, nb2 = 0u;
                        auto near_pair = [&](uint32_t p, uint32_t &nb) {
                            const float4 A = rp[2 * p], Bz = rp[2 * p + 1];
                            const float2 d0 = __fadd2_rn(make_float2(A.x, A.y), nx[k]), d1 = __fadd2_rn(make_float2(A.z, A.w), ny[k]);
                            float2 nH = nHs2_u, tl = make_float2(tol_u, tol_u);
                            if (VARH) {
                                const float2 Hs = __fmul2_rn(make_float2(fmaxf(Bz.z, hj[k]), fmaxf(Bz.w, hj[k])),
                                                             make_float2(sp.scale, sp.scale));
                                nH = __fmul2_rn(Hs, make_float2(-Hs.x, -Hs.y));
                                tl = __fmul2_rn(make_float2(-nH.x, -nH.y), make_float2(band, band));
                            }
                            float2 acc = __ffma2_rn(d0, d0, nH);
                            acc = __ffma2_rn(d1, d1, acc);
                            if (DIM == 3) {
                                const float2 d2 = __fadd2_rn(make_float2(Bz.x, Bz.y), nz[k]);
                                acc = __ffma2_rn(d2, d2, acc);
                            }
                            nb = (nb << 2) | (fabsf(acc.x) <= tl.x ? 2u : 0u) | (fabsf(acc.y) <= tl.y ? 1u : 0u);
                        };
                        for (uint32_t p = 0; p < np1; ++p) near_pair(p, nb1);
                        for (uint32_t p = 0; p < np2; ++p) near_pair(16u + p, nb2);
                        if (!flagged) continue;
                        const float4 pj_orig = pos_s[tile_q_to_sorted(tt, qk[k])];
                        while (nb1 | nb2) {
                            const bool first = nb1 != 0u;
                            const uint32_t bit = 31u - (uint32_t)__clz(first ? nb1 : nb2);
                            if (first) nb1 ^= 1u << bit; else nb2 ^= 1u << bit;
                            const uint32_t i = first ? 2u * np1 - 1u - bit : 32u + 2u * np2 - 1u - bit;
                            if (i >= nr) continue;                              // the duplicate of an odd last row
                            const uint32_t local = r_lo + i;
                            const float4 pi_orig = pos_s[tt.h_start[hc_i] + local];
                            const float Hs = VARH ? __fmul_rn(sp.scale, fmaxf(pi_orig.w, pj_orig.w)) : sp.Hs_u;
                            const uint32_t hit = pred_exact(pi_orig, pj_orig, Hs, gg) ? 1u : 0u;
                            if (first) rb[k] = (rb[k] & ~(1u << bit)) | (hit << bit);
                            else rb2[k] = (rb2[k] & ~(1u << bit)) | (hit << bit);
                        }
                    }
                    // first word: transpose -- lane b receives the mask of row slot i = b - (32 - 2 np1), candidate c at
                    // bit 31 - c.  Second word: likewise when it holds many rows, else one ballot per row.
                    const uint32_t row_base = c_rb[tc] + r_lo;
                    const int islot = lane - (32 - 2 * (int)np1), islot2 = lane - (32 - 2 * (int)np2);
#pragma unroll
                    for (int k = 0; k < kCPL; ++k) {
                        const uint32_t w = cb * kCPL + k;
                        if (w * 32u >= Nc) continue;                       // uniform: no valid candidate in this word
                        SPH_ASSERT(w < (uint32_t)fs.wcap && row_base + nr <= (uint32_t)tcap);
                        uint32_t *mw = sm.masks + (size_t)w * tcap + row_base;
                        // rows i < nr1 sit at bits 2 np1 - 1 - i (the duplicate of an odd last row below them is not a row)
                        my_hits += (uint32_t)__popc(rb[k] >> (2u * np1 - nr1)) + (nr2 ? (uint32_t)__popc(rb2[k] >> (2u * np2 - nr2)) : 0u);
                        const uint32_t y = warp_transpose32(rb[k]);
                        if (islot >= 0 && (uint32_t)islot < nr1) mw[islot] = y;
                        if (nr2 > 8u) {
                            const uint32_t y2 = warp_transpose32(rb2[k]);
                            if (islot2 >= 0 && (uint32_t)islot2 < nr2) mw[32 + islot2] = y2;
                        } else {
                            for (uint32_t i2 = 0; i2 < nr2; ++i2) {
                                const uint32_t v = __brev(__ballot_sync(0xffffffffu, (rb2[k] >> (2u * np2 - 1u - i2)) & 1u));
                                if (lane == 0) mw[32u + i2] = v;
                            }
                        }
                    }
                }
        }
        my_hits = __reduce_add_sync(0xffffffffu, my_hits);
        if (lane == 0 && my_hits) atomicAdd(&s_hits, my_hits);
    }
    __syncthreads();                                          // masks complete, s_hits = entries of the tile

    // ---- phase 2: warp 0 looks back for the tile's base (its total is known already) WHILE the other warps count the
    // rows, split them for phase 3 and scan the counts; they meet at a barrier of their own, warp 0 joins phase 3 when the
    // base is there.
    const uint32_t tot = s_hits;
    if (warp == 0) {
        const long long b = tile_lookback(tstate, ticket, tot);
        if (lane == 0) {
            s_base = b;
            __threadfence_block();
            s_ready = 1u;
        }
    } else {
    const uint32_t nthr2 = blockDim.x - 32u;
    for (uint32_t r = threadIdx.x - 32u; r < T; r += nthr2) {
        // the row's mask words are split among its four lanes of phase 3 at word boundaries, by HITS (the words of the
        // middle plane of the neighbourhood hold twice the hits of the outer ones): lane q starts at the first word at
        // which the running count reaches q/4 of the total
        const uint32_t Wc = (c_nc[sm.rowcell[r]] + 31u) >> 5;
        uint32_t c = 0;
        for (uint32_t w = 0; w < Wc; ++w) c += (uint32_t)__popc(sm.masks[(size_t)w * tcap + r]);
        {
            uint32_t run = 0, q = 1;
            for (uint32_t w = 0; w < Wc && q < 4u; ++w) {
                while (q < 4u && 4u * run >= q * c) {
                    sm.qcnt[3 * r + q - 1u] = (uint16_t)run;
                    sm.qwrd[3 * r + q - 1u] = (uint8_t)w;
                    ++q;
                }
                run += (uint32_t)__popc(sm.masks[(size_t)w * tcap + r]);
            }
            for (; q < 4u; ++q) {
                sm.qcnt[3 * r + q - 1u] = (uint16_t)c;
                sm.qwrd[3 * r + q - 1u] = (uint8_t)Wc;
            }
        }
        sm.off[r] = c;
    }
    asm volatile("bar.sync 1, %0;" ::"r"(nthr2) : "memory");    // warps 1 .. kFW-1: counts complete
    if (warp == 1) {
        uint32_t carry = 0;
        for (uint32_t r0 = 0; r0 < T; r0 += 32) {
            const uint32_t r = r0 + lane;
            const uint32_t c = r < T ? sm.off[r] : 0u;
            uint32_t inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (r < T) sm.off[r] = carry + inc - c;
            carry += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) {
            sm.off[T] = carry;
            s_tot = carry;
        }
        __syncwarp();
        if (lane == 0) {
            SPH_ASSERT(s_tot == tot);
            __threadfence_block();
            s_off_ready = 1u;
        }
    }
    asm volatile("bar.sync 1, %0;" ::"r"(nthr2) : "memory");    // off[] complete for the warps that wrote it
    }
    if (warp == 0) {
        while (s_off_ready == 0u) __nanosleep(100);
        __threadfence_block();
    }

    // ---- phase 3: masks -> halo indices.  Groups of 8 consecutive rows, handed out to the warps by a shared counter; a
    // warp expands a group into its own image (four lanes per row, each a quarter of the row's mask words, one flat
    // predicated loop) -- that needs no base, so the warps do it while warp 0 is still looking back -- then waits for
    // the base and flushes with 16-byte stores.
    constexpr uint32_t kGR = 32 / kRowLanes;                     // rows of a group
    const uint32_t wcap = (((uint32_t)fs.scap + 8u) / (uint32_t)kFW - 8u) & ~7u;   // entries of a warp's image (+ 8 of slack)
    uint16_t *wst = sm.stage + (size_t)warp * (wcap + 8u);
    SPH_ASSERT((size_t)kFW * (wcap + 8u) <= (size_t)fs.scap + 8u);
    const uint32_t mstride = (uint32_t)tcap * 4u;
    const uint32_t ngroups = (T + kGR - 1u) / kGR;
    long long base = -1;
    for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = atomicAdd(&s_grp, 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= ngroups) break;
        const uint32_t ra = g * kGR, rb = min(T, ra + kGR);
        const uint32_t total = sm.off[rb] - sm.off[ra];
        const bool direct = total > wcap;                       // dense rows: straight to global memory
        const uint32_t r = min(ra + (uint32_t)lane / kRowLanes, T - 1u), part = (uint32_t)lane % kRowLanes;
        const bool live = ra + (uint32_t)lane / kRowLanes < rb;
        const uint32_t tc = sm.rowcell[r];
        const uint32_t Wc = (c_nc[tc] + 31u) >> 5;
        const uint32_t w0 = part ? (uint32_t)sm.qwrd[3 * r + part - 1u] : 0u;
        const uint32_t w1 = live ? (part < 3u ? (uint32_t)sm.qwrd[3 * r + part] : Wc) : w0;
        const uint32_t o = sm.off[r] - sm.off[ra] + (part ? (uint32_t)sm.qcnt[3 * r + part - 1u] : 0u);
        if (!direct) {
            uint32_t maddr = (uint32_t)__cvta_generic_to_shared(sm.masks + (size_t)w0 * tcap + r);
            const uint32_t mend = maddr + (w1 - w0) * mstride;
            uint32_t cnext = (uint32_t)__cvta_generic_to_shared(sm.cmap + (size_t)tc * ncap + 32u * w0) + 62u;
            uint32_t ccur = cnext;
            uint32_t daddr = (uint32_t)__cvta_generic_to_shared(wst + 8u + o);
            uint32_t m = 0, vpend = 0, pend = 0;
            // One predicated block per step: a lane whose word is empty fetches its next word, any other lane emits its
            // highest set bit (= lowest candidate).  The candidate-map load of a hit is consumed one step later (the
            // store of the PREVIOUS hit goes first), so its latency does not sit in the chain.  Two steps per vote.
            for (;;) {
#pragma unroll
                for (int rep = 0; rep < 2; ++rep)
                    asm volatile(
                        "{\n"
                        ".reg .pred pe, pf, pp;\n"
                        ".reg .u32 hb, bit, ca;\n"
                        "setp.ne.u32 pp, %6, 0;\n"
                        "@pp st.shared.u16 [%3], %5;\n"
                        "@pp add.u32 %3, %3, 2;\n"
                        "setp.eq.u32 pe, %0, 0;\n"
                        "setp.ne.and.u32 pf, %2, %8, pe;\n"
                        "selp.u32 %6, 0, 1, pe;\n"
                        "@!pe bfind.u32 hb, %0;\n"
                        "@!pe shl.b32 bit, 1, hb;\n"
                        "@!pe xor.b32 %0, %0, bit;\n"
                        "@!pe shl.b32 hb, hb, 1;\n"
                        "@!pe sub.u32 ca, %1, hb;\n"
                        "@!pe ld.shared.u16 %5, [ca];\n"
                        "@pf ld.shared.u32 %0, [%2];\n"
                        "@pf mov.u32 %1, %4;\n"
                        "@pf add.u32 %2, %2, %7;\n"
                        "@pf add.u32 %4, %4, 64;\n"
                        "}\n"
                        : "+r"(m), "+r"(ccur), "+r"(maddr), "+r"(daddr), "+r"(cnext), "+r"(vpend), "+r"(pend)
                        : "r"(mstride), "r"(mend)
                        : "memory");
                if (__all_sync(0xffffffffu, m == 0u && maddr == mend && pend == 0u)) break;
            }
            SPH_ASSERT(daddr <= (uint32_t)__cvta_generic_to_shared(wst + 8u + wcap));        // the warp's image was not overrun
        }
        if (base < 0) {                                          // first group of this warp: the base may still be on its way
            while (s_ready == 0u) __nanosleep(200);           // leave the issue slots to the warps that still expand
            __threadfence_block();
            base = s_base;
            if (base + (long long)tot > fs.col_cap) {             // uniform per CTA: every warp takes this exit
                if (threadIdx.x == 0) atomicOr(&ctl[1], 1u);
                base = -2;
            }
        }
        // offsets and counts of the group's rows (exact even when the lists do not fit)
        if ((uint32_t)lane < kGR && ra + lane < rb) {
            const long long bb = base >= 0 ? base : s_base;
            row_ptr[tt.row0 + ra + lane] = bb + sm.off[ra + lane];
            cnt_out[tt.row0 + ra + lane] = sm.off[ra + lane + 1] - sm.off[ra + lane];
            if (ra + lane + 1 == T && (long long)tt.row0 + T == n) row_ptr[n] = bb + tot;
        }
        if (base == -2) continue;
        const long long g0 = base + sm.off[ra];                  // first entry of the group in col16
        if (!direct) {
            __syncwarp();
            // global vector v holds entries 8 v - gsh ... 8 v - gsh + 7 of the group (image index + 8)
            const uint32_t gsh = (uint32_t)(g0 & 7ll);
            uint4 *gv = reinterpret_cast<uint4 *>(col16 + (g0 - gsh));
            const uint32_t nvec = (gsh + total + 7u) >> 3;
            for (uint32_t v = lane; v < nvec; v += 32) {
                const int j0 = (int)(8u * v) - (int)gsh;
                if (j0 >= 0 && j0 + 8 <= (int)total) {
                    const uint16_t *e = wst + 8 + j0;
                    uint4 val;
                    val.x = (uint32_t)e[0] | ((uint32_t)e[1] << 16);
                    val.y = (uint32_t)e[2] | ((uint32_t)e[3] << 16);
                    val.z = (uint32_t)e[4] | ((uint32_t)e[5] << 16);
                    val.w = (uint32_t)e[6] | ((uint32_t)e[7] << 16);
                    gv[v] = val;
                } else {
                    for (int k = 0; k < 8; ++k)
                        if (j0 + k >= 0 && j0 + k < (int)total) col16[g0 + j0 + k] = wst[8 + j0 + k];
                }
            }
            __syncwarp();
        } else if (live) {
            uint16_t *dst = col16 + g0 + o;
            const uint16_t *cm = sm.cmap + (size_t)tc * ncap;
            uint32_t k = 0;
            for (uint32_t w = w0; w < w1; ++w) {
                uint32_t m = sm.masks[(size_t)w * tcap + r];
                while (m) {
                    const int hb = 31 - __clz(m);
                    m ^= 1u << hb;
                    SPH_ASSERT(32u * w + 31u - (uint32_t)hb < (uint32_t)ncap);
                    dst[k++] = cm[32u * w + 31u - (uint32_t)hb];
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------- cell statistics
// out[0] = largest number of candidates of a cell (particles of its 3^d neighbour cells), out[2..3] = sum over all rows
// of their candidate counts (a hard upper bound of nnz), one thread per cell
template <int DIM>
__global__ void k_cell_stats(GridGeom gg, long long ncells, const uint32_t *__restrict__ cell_start,
                             const uint32_t *__restrict__ cell_end, uint32_t *__restrict__ out)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t nc = 0;
    unsigned long long pairs = 0;
    if (c < ncells) {
        int cc[3];
        long long t = c;
        cc[0] = (int)(t % gg.ncell[0]); t /= gg.ncell[0];
        cc[1] = (int)(t % gg.ncell[1]); t /= gg.ncell[1];
        cc[2] = (int)t;
        const uint32_t own = cell_end[c] - cell_start[c];
        if (own) {
            const int zlo = DIM == 3 ? -1 : 0, zhi = DIM == 3 ? 1 : 0;
            for (int dz = zlo; dz <= zhi; ++dz)
                for (int dy = -1; dy <= 1; ++dy)
                    for (int dx = -1; dx <= 1; ++dx) {
                        int q[3] = {cc[0] + dx, cc[1] + dy, cc[2] + dz};
                        bool ok = true;
#pragma unroll
                        for (int k = 0; k < DIM; ++k) {
                            if (gg.periodic[k]) q[k] = q[k] < 0 ? q[k] + gg.ncell[k] : (q[k] >= gg.ncell[k] ? q[k] - gg.ncell[k] : q[k]);
                            else if (q[k] < 0 || q[k] >= gg.ncell[k]) ok = false;
                        }
                        if (!ok) continue;
                        const long long lin = ((long long)q[2] * gg.ncell[1] + q[1]) * gg.ncell[0] + q[0];
                        nc += cell_end[lin] - cell_start[lin];
                    }
            pairs = (unsigned long long)own * nc;
        }
    }
    nc = __reduce_max_sync(0xffffffffu, nc);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) pairs += __shfl_xor_sync(0xffffffffu, pairs, o);
    if ((threadIdx.x & 31) == 0) {
        if (nc) atomicMax(&out[0], nc);
        if (pairs) atomicAdd(reinterpret_cast<unsigned long long *>(out + 2), pairs);
    }
}

} // namespace

// enqueue the cell statistics the fused build sizes itself with (read back with the other statistics of sph_neighbors)
int sph_fused_stats_launch(sph_ctx *ctx, cudaStream_t st)
{
    SPH_TRY(ctx->fstats.reserve(64));
    SPH_CUDA_TRY(cudaMemsetAsync(ctx->fstats.p, 0, 16, st));
    const GridGeom &gg = ctx->geom;
    const long long nc = ctx->ncells_total;
    KScope ks(ctx, SPH_K_COUNT, 1, st);
    const unsigned nb = (unsigned)((nc + 127) / 128);
    if (gg.dim == 3) k_cell_stats<3><<<nb, 128, 0, st>>>(gg, nc, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), ctx->fstats.as<uint32_t>());
    else k_cell_stats<2><<<nb, 128, 0, st>>>(gg, nc, ctx->cell_start.as<uint32_t>(), ctx->cell_end.as<uint32_t>(), ctx->fstats.as<uint32_t>());
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

// Tiles in the order of their rows in the sorted arrays: the sort key is the Morton code of the cell, a tile is an aligned
// block of B^d cells with B a power of two, so tile (bx,by,bz) holds the keys whose high bits are the Morton code of
// (bx,by,bz).  Depends on the grid only; rebuilt when the grid or B changes.
static int fused_tile_order(sph_ctx *ctx, const TileGeom &tg, cudaStream_t st)
{
    for (auto &slot : ctx->tile_orders)
        if (slot.valid && slot.B == tg.B && slot.dim == tg.dim && slot.nb[0] == tg.nb[0] && slot.nb[1] == tg.nb[1] &&
            slot.nb[2] == tg.nb[2]) {
            ctx->tile_order_cur = slot.buf.as<uint32_t>();
            return SPH_OK;
        }
    // (a step that alternates between two grids, like bench.py's, keeps both orders)
    auto &slot = ctx->tile_orders[ctx->tile_order_next];
    ctx->tile_order_next = (ctx->tile_order_next + 1) % 4;
    slot.valid = false;
    std::vector<std::pair<uint64_t, uint32_t>> keys((size_t)tg.ntiles);
    for (int t = 0; t < tg.ntiles; ++t) {
        int b = t;
        const uint32_t bx = (uint32_t)(b % tg.nb[0]);
        b /= tg.nb[0];
        const uint32_t by = (uint32_t)(b % tg.nb[1]), bz = (uint32_t)(b / tg.nb[1]);
        uint64_t k = 0;
        for (int bit = 0; bit < 20; ++bit) {
            if (tg.dim == 3)
                k |= ((uint64_t)((bx >> bit) & 1u) << (3 * bit)) | ((uint64_t)((by >> bit) & 1u) << (3 * bit + 1)) |
                     ((uint64_t)((bz >> bit) & 1u) << (3 * bit + 2));
            else
                k |= ((uint64_t)((bx >> bit) & 1u) << (2 * bit)) | ((uint64_t)((by >> bit) & 1u) << (2 * bit + 1));
        }
        keys[(size_t)t] = {k, (uint32_t)t};
    }
    std::sort(keys.begin(), keys.end());
    ctx->tile_order_host.resize((size_t)tg.ntiles);
    for (int t = 0; t < tg.ntiles; ++t) ctx->tile_order_host[(size_t)t] = keys[(size_t)t].second;
    SPH_TRY(slot.buf.reserve((size_t)tg.ntiles * 4));
    // pageable source: the copy is staged before the call returns, so the vector may be reused afterwards
    SPH_CUDA_TRY(cudaMemcpyAsync(slot.buf.p, ctx->tile_order_host.data(), (size_t)tg.ntiles * 4, cudaMemcpyHostToDevice, st));
    slot.valid = true;
    slot.B = tg.B;
    slot.dim = tg.dim;
    for (int k = 0; k < 3; ++k) slot.nb[k] = tg.nb[k];
    ctx->tile_order_cur = slot.buf.as<uint32_t>();
    return SPH_OK;
}

// Count, offsets and fill of the tile-local lists with tile edge B in one kernel.  Returns 1 when a tile does not fit
// the kernel's shared-memory carve-up (the caller then takes the two-kernel build).  Synchronises `st` once.
int sph_neighbors_fused_run(sph_ctx *ctx, const SearchPar &sp, const TileGeom &tg, uint32_t Mmax, uint32_t Tmax,
                            uint32_t ncmax, unsigned long long pairs_bound, cudaStream_t st, int64_t *nnz_out)
{
    const int64_t n = ctx->n;
    const GridGeom &gg = ctx->geom;
    const bool varh = ctx->hmin != ctx->hmax;
    const int warps = ctx->opt_fused_warps ? ctx->opt_fused_warps : kFWmax;
    FusedSizes fs;
    fs.mcap = (int)((Mmax + 7u) & ~7u);
    fs.tcap = (int)((Tmax + 7u) & ~7u);
    fs.ncap = (int)((ncmax + kCandBlock - 1) / kCandBlock * kCandBlock);
    if (fs.ncap < kCandBlock) fs.ncap = kCandBlock;
    fs.wcap = (int)((ncmax + 31u) / 32u);
    if (fs.wcap < 1) fs.wcap = 1;
    fs.nt_max = 1;
    for (int k = 0; k < gg.dim; ++k) fs.nt_max *= tg.B;
    fs.pcap = fs.tcap / 2 + fs.nt_max + 1;
    if (Mmax == 0 || Mmax >= kQNone || fs.nt_max > kTileMaxTgt || fs.ncap / 32 > 255) return 1;
    // entries per row: the last build's mean if there was one, else a fraction of the candidates (ball / cube of cells)
    double mean_len;
    if (ctx->nnz > 0 && ctx->n_lists == n && ctx->search_scale > 0.f)
        mean_len = (double)ctx->nnz / (double)n * pow((double)sp.scale / (double)ctx->search_scale, gg.dim);
    else mean_len = (double)pairs_bound / (double)n * (gg.dim == 3 ? 0.20 : 0.42);
    if (mean_len < 1.0) mean_len = 1.0;
    const size_t r0 = (size_t)fs.mcap * 16 + (size_t)fs.pcap * 32;
    fs.scap = 8;
    const size_t fixed = fused_fixed_bytes(fs) + 16;
    // 227 KB per CTA minus the kernel's static shared memory (asked from the runtime, largest of the four variants)
    static size_t static_smem = 0;
    if (!static_smem) {
        cudaFuncAttributes fa;
        size_t mx = 0;
        SPH_CUDA_TRY(cudaFuncGetAttributes(&fa, k_nb_fused<2, false>)); mx = std::max(mx, fa.sharedSizeBytes);
        SPH_CUDA_TRY(cudaFuncGetAttributes(&fa, k_nb_fused<2, true>)); mx = std::max(mx, fa.sharedSizeBytes);
        SPH_CUDA_TRY(cudaFuncGetAttributes(&fa, k_nb_fused<3, false>)); mx = std::max(mx, fa.sharedSizeBytes);
        SPH_CUDA_TRY(cudaFuncGetAttributes(&fa, k_nb_fused<3, true>)); mx = std::max(mx, fa.sharedSizeBytes);
        static_smem = (mx + 127) & ~(size_t)127;
    }
    const size_t cta_max = 232448 - static_smem, two = (233472 - 2 * 5120) / 2;   // two CTAs per SM: 1 KB each set aside
    if (fixed + r0 > cta_max) return 1;
    const size_t budget = fixed + r0 <= two ? two : cta_max;
    {
        // staging: one image of 32 / kRowLanes rows per warp (+ 8 entries of slack each); longer groups go straight to global memory
        const double want = (double)warps * ((32.0 / kRowLanes) * mean_len * 1.35 + 48.0);
        size_t room = (budget - fixed) / 2 - 16;                      // entries
        size_t sc = want < (double)room ? (size_t)want : room;
        if (sc * 2 + 16 < r0) sc = (r0 - 16) / 2;                     // the overlay region is there anyway
        fs.scap = (int)(sc & ~(size_t)7);
    }
    const size_t smem = fused_smem_bytes(fs);
    SPH_TRY(ctx->cnt.reserve((size_t)n * 4));
    SPH_TRY(ctx->row_ptr.reserve((size_t)(n + 1) * 8));
    SPH_TRY(ctx->tstate.reserve((size_t)tg.ntiles * 8));
    SPH_TRY(ctx->fctl.reserve(16));
    SPH_TRY(fused_tile_order(ctx, tg, st));
    // capacity of col16: never shrinks; first guess from the same estimate, exact on the (rare) second attempt
    {
        double guess = (double)n * mean_len * 1.1 + 4096.0;
        if (guess > (double)pairs_bound + 64.0) guess = (double)pairs_bound + 64.0;
        SPH_TRY(ctx->col16.reserve((size_t)guess * 2 + 64));
    }
    int64_t nnz = 0;
    for (int attempt = 0; attempt < 2; ++attempt) {
        fs.col_cap = (long long)(ctx->col16.cap / 2) - 16;
        SPH_CUDA_TRY(cudaMemsetAsync(ctx->tstate.p, 0, (size_t)tg.ntiles * 8, st));
        SPH_CUDA_TRY(cudaMemsetAsync(ctx->fctl.p, 0, 16, st));
        {
            KScope ks(ctx, SPH_K_FILL, 1, st);
#define SPH_NBF_LAUNCH(DIM, VARH)                                                                                      \
    do {                                                                                                               \
        SPH_CUDA_TRY(cudaFuncSetAttribute(k_nb_fused<DIM, VARH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        k_nb_fused<DIM, VARH><<<(unsigned)tg.ntiles, warps * 32, smem, st>>>(                                            \
            tg, gg, sp, fs, (long long)n, ctx->pos_s.as<float4>(), ctx->cell_start.as<uint32_t>(),                     \
            ctx->cell_end.as<uint32_t>(), ctx->tile_order_cur, ctx->fctl.as<uint32_t>(),                    \
            ctx->tstate.as<unsigned long long>(), ctx->cnt.as<uint32_t>(), ctx->row_ptr.as<long long>(),               \
            ctx->col16.as<uint16_t>());                                                                                \
    } while (0)
            if (gg.dim == 3) { if (varh) SPH_NBF_LAUNCH(3, true); else SPH_NBF_LAUNCH(3, false); }
            else { if (varh) SPH_NBF_LAUNCH(2, true); else SPH_NBF_LAUNCH(2, false); }
#undef SPH_NBF_LAUNCH
        }
        SPH_CUDA_TRY(cudaGetLastError());
        SPH_CUDA_TRY(cudaMemcpyAsync(ctx->h_pinned + 4, ctx->row_ptr.as<long long>() + n, 8, cudaMemcpyDeviceToHost, st));
        SPH_CUDA_TRY(cudaMemcpyAsync(ctx->h_pinned + 5, ctx->fctl.as<uint32_t>() + 1, 4, cudaMemcpyDeviceToHost, st));
        SPH_CUDA_TRY(cudaStreamSynchronize(st));
        nnz = ctx->h_pinned[4];
        uint32_t over = 0;
        memcpy(&over, ctx->h_pinned + 5, 4);
        if (!over) break;
        if (attempt == 1) return SPH_E_CUDA;                           // cannot happen: the capacity was exact
        SPH_TRY(ctx->col16.reserve((size_t)nnz * 2 + 64));
    }
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

#ifdef SPH_BOUNDS
unsigned int sph_bounds_read_fused()
{
    unsigned int v = 0;
    cudaMemcpyFromSymbol(&v, sph_bounds_count, sizeof(v));
    return v;
}
#endif
