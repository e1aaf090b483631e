// sph_internal.cuh -- context, scratch arena and small device helpers shared by the sm_100a kernels.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <vector>

#include "../../include/sph.h"

#define SPH_CUDA_TRY(expr)                                   \
    do {                                                     \
        cudaError_t e__ = (expr);                            \
        if (e__ != cudaSuccess) {                            \
            (void)cudaGetLastError();                        \
            return e__ == cudaErrorMemoryAllocation ? SPH_E_NOMEM : SPH_E_CUDA; \
        }                                                    \
    } while (0)

#define SPH_TRY(expr)               \
    do {                            \
        int r__ = (expr);           \
        if (r__ != SPH_OK) return r__; \
    } while (0)

// One device buffer that only ever grows.
struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    int reserve(size_t bytes)
    {
        if (bytes <= cap) return SPH_OK;
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
        size_t want = bytes + bytes / 16 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            p = nullptr;
            return SPH_E_NOMEM;
        }
        cap = want;
        return SPH_OK;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
    template <class T> T *as() const { return reinterpret_cast<T *>(p); }
};

// Geometry of the cell grid as the kernels see it (passed by value).
struct GridGeom {
    int dim;
    int periodic[3];
    int ncell[3];
    int bits;          // Morton bits per axis
    float lo[3], hi[3];
    float L[3];        // binary32 hi - lo (the one L of the readings R3/R4)
    double lo_d[3];
    double edge[3];    // cell edge per axis (binary64)
    double L_d[3];
};

// Cell-block decomposition (sph_tiles.cuh); passed by value.
struct TileGeom {
    int dim;
    int B;             // block edge in cells: 1, 2 or 4
    int nb[3];         // blocks per axis
    int ntiles;
    int ncell[3];
    int periodic[3];
    float L[3];
    const void *tabs;  // device TileTab[ntiles] written once per build (k_tile_tables), or NULL: every CTA derives its own
};

// Per-launch physical constants (derived once on the host from sph_params).
struct KPar {
    int dim;
    int periodic[3];
    float L[3], halfL[3], lo[3], hi[3];
    float c0, rho0, gamma, delta, alpha, nu, eps;
    float g[3];
    float Cd;       // kernel normalisation C_d
    float inv_kappa; // 1/kappa_d
    float visc_nu;  // 2(d+2) nu
    float Bp;       // rho0 c0^2 / gamma
    int form;       // pressure form: 0 symmetric Eq.40, 1 (p_i+p_j)/(rho_i rho_j)
    int delta_form; // 0 Molteni-Colagrossi delta-term, 1 with the renormalised density gradient of [43]
    float rcond;    // eigenvalue cutoff of the pseudo-inverse L_i (delta_form 1)
    int uniform_h;  // all h equal (then the H-dependent constants below are valid)
    float H, invH, cW, cG, cK, ell, e2, eta, kd;
};

// Optional per-kernel-class device timing (sph_profile_enable / sph_profile_read): a pair of CUDA events on the
// launching stream around every launch (or group of launches) of a class, resolved when read.
struct ProfRec {
    cudaEvent_t a, b;
    int cls;
};
struct Profiler {
    bool on = false;
    std::vector<ProfRec> live;                                  // recorded, not yet resolved
    std::vector<cudaEvent_t> pool;                              // free events
    double ms[SPH_K_NCLASS] = {0};
    int64_t count[SPH_K_NCLASS] = {0};
    cudaEvent_t get()
    {
        if (!pool.empty()) {
            cudaEvent_t e = pool.back();
            pool.pop_back();
            return e;
        }
        cudaEvent_t e = nullptr;
        cudaEventCreate(&e);
        return e;
    }
};

struct sph_ctx {
    int device = 0;
    Profiler prof;
    int opt_group = 0;          // lanes per row in the pair kernels (0 = default)
    int opt_warps = 0;          // warps per CTA of the tile pair kernels (0 = automatic: 8, or 16 when one CTA fits an SM)
    int opt_list_mode = 0;      // 0 auto, 1 force the generic (global-id) lists, 2 force tile-local lists
    int opt_rk_extra_permille = -1;  // sph_rk_step: extra list skin (1/1000 of h) that lets later steps reuse the lists;
                                     // -1 = automatic (2D: whatever the cell size leaves, capped; 3D: none)
    float scale_slack_cap = 0.f;     // set by sph_rk_step around its sph_neighbors call: the search scale may grow by up to
                                     // this much if the cell size allows
    sph_domain dom_last{};      // domain of the last sph_build_cells
    int opt_fill_masks = 1;     // the fill expands the hit masks saved by the count pass (0: repeats the tests)
    int opt_tile_edge = 0;      // 0 auto, else force the tile edge B (1, 2, 4)
    int opt_fused_warps = 0;    // warps per CTA of the one-kernel build (0 = default)
    int opt_build_fused = 1;    // 1: the tile-local lists are built by the one-kernel build (sph_neighbors_fused.cu) when a tile fits it
    int opt_stage_bulk = 0;     // 1: k_rhs_tile / k_vjp_tile stage their float4 halo arrays with cp.async.bulk + one mbarrier (measured: profiles/r02_f)
    int opt_tile_tables = 1;    // 1: the tables of a tile are computed once per build and loaded by the tile kernels
    int opt_vjp_split = 1;      // 1: k_vjp_tile works on half a 2x2x2 tile per CTA (two resident CTAs per SM instead of one)
    int opt_no_um = 0;          // 1: never launch the uniform-mass variants of the tile pair kernels (A/B measurements, tests)
    bool tile_mode = false;     // lists of the last sph_neighbors are tile-local (col16)
    TileGeom tg{};
    uint32_t tile_Mmax = 0, tile_Tmax = 0;   // largest halo / row count of a tile
    uint32_t tile_Mhalf = 0;                 // largest halo of HALF a tile (3D, 2x2x2 cells: three z-layers); 0 = no halves
    int64_t n_hint = 0;
    int64_t n = 0;
    bool cells_ready = false, lists_ready = false;
    GridGeom geom{};
    int64_t ncells_total = 0;
    float search_scale = 1.f;
    int64_t nnz = 0;
    int64_t launches = 0;
    cudaStream_t last_stream = nullptr;
    float hmin = 0.f, hmax = 0.f;

    // cells / sort
    DevBuf key_a, key_b, idx_a, idx_b, hist;
    DevBuf perm, inv_perm;      // sorted -> caller, caller -> sorted
    DevBuf key_sorted;          // alias target of the last sort pass (copy)
    DevBuf pos_s;               // float4 {xw,yw,zw,h} at build time, sorted
    DevBuf cell_start, cell_end;
    DevBuf stats;               // device: [0] err flag, [1] hmax bits, [2] hmin bits
    // lists
    DevBuf cnt, row_ptr, col, col16, scan_tmp;
    DevBuf maskbuf, tile_words, tile_mask_base;   // hit masks of the count pass, per-tile mask offsets
    // one-kernel build: cell statistics, look-back states, {ticket, overflow}, tiles in Morton order (cached per grid)
    DevBuf fstats, tstate, fctl;
    DevBuf tile_tabs;           // TileTab of every tile of the last build (sph_tiles.cuh)
    const float4 *pos_override = nullptr;         // sph_shift: sph_grad_sum's kernels read these positions instead of pos_s
    // delta_form 1: current positions {x,y,z,h}, {V,rho}, moments, {g,V}, adjoint records and sorted partial results
    DevBuf d_pos, d_va, d_mom, d_g4, d_lr, d_dx4, d_gb4, d_rb, d_rc, d_rd, d_re, d_x2, d_vb, d_ab, d_part;
    struct TileOrder {                            // cache slot: the order depends on the grid and on B only
        DevBuf buf;
        bool valid = false;
        int B = 0, dim = 0, nb[3] = {0, 0, 0};
    } tile_orders[4];
    int tile_order_next = 0;                      // slot replaced next
    const uint32_t *tile_order_cur = nullptr;     // order of the current build (device)
    std::vector<uint32_t> tile_order_host;
    uint32_t f_ncmax = 0;                         // largest candidate count of a cell (k_cell_stats)
    unsigned long long f_pairs = 0;               // sum over rows of their candidate counts: upper bound of nnz
    int64_t n_lists = 0;                          // n of the lists `nnz` belongs to
    bool col_valid = false;     // ctx->col holds the global-id lists of the current build
    // pair scratch (sorted SoA)
    DevBuf s0, s1, s2, s3, c0buf, out4, m_s, kind_s, partials, eos;
    // rk scratch
    DevBuf rk[16];
    // pinned host mirror
    int64_t *h_pinned = nullptr; // [16]
    // sph_step_host: copies that are not on the critical path run on their own stream
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_in = nullptr, ev_out = nullptr;
    // sph_step_host: the final update of sph_rk_step runs in `rk_final_chunks` ranges of caller indices, each followed by
    // an event, so that the device-to-host copy of one range overlaps the update of the next
    int rk_final_chunks = 1;
    bool rk_lists_prepared = false;  // sph_step_host has already run sph_rk_prepare_lists for the coming sph_rk_step
    cudaEvent_t ev_final[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_final_x = nullptr;     // sph_step_host: the advanced positions are complete (before the last RHS)
    // host staging for *_host call
    DevBuf hx, hv, hrho, hm, hh, hkind, hlam, hmu, ho_drho, ho_acc, ho_xb, ho_vb, ho_rb, ho_pb, ho_dens;
};

// device flag pair of the uniform-mass fast path: [0] non-zero = all masses of the last pack equal, [1] = that mass
// (float bits).  Written on the stream by the pack kernels (k_pack_state, k_rk_base), read by the pair kernels: the
// host never needs to know -- both variants of a pair kernel are launched and the one whose turn it is not returns.
constexpr int kUmSlot = 13;
constexpr int kDensUmSlot = 3;        // stats word: all masses of the last sph_density call are equal (its own gather kernel writes it)
constexpr int kTileHalfSlot = 15;      // stats word: largest halo of half a 2x2x2 tile (three of its four z-layers of cells)
inline uint32_t *sph_um_flag(const sph_ctx *ctx) { return ctx->stats.as<uint32_t>() + kUmSlot; }
#ifdef __CUDACC__
// Pack kernels: a density that is not a positive finite number, or a mass that is not finite, raises bit 4 of the
// sticky device error flag (stats[0], the word k_wrap_key uses for positions and h; `um` points kUmSlot words past it).
// Reported as SPH_E_DOMAIN by the next synchronising call or sph_check.
__device__ __forceinline__ void sph_flag_bad_state(uint32_t *um, float rho, float m)
{
    if (!(rho > 0.f && rho <= 3.402823466e38f) || !(fabsf(m) <= 3.402823466e38f)) atomicOr(um - kUmSlot, 4u);
}
#endif

// Counts `nlaunch` kernel launches of class `cls` and, when profiling is on, brackets them with events on `st`.
struct KScope {
    sph_ctx *ctx;
    cudaStream_t st;
    ProfRec rec{};
    bool timed;
    KScope(sph_ctx *c, int cls, int nlaunch, cudaStream_t s) : ctx(c), st(s), timed(c->prof.on)
    {
        ctx->launches += nlaunch;
        ctx->prof.count[cls] += nlaunch;
        if (timed) {
            rec.a = ctx->prof.get();
            rec.b = ctx->prof.get();
            rec.cls = cls;
            cudaEventRecord(rec.a, st);
        }
    }
    ~KScope()
    {
        if (timed) {
            cudaEventRecord(rec.b, st);
            ctx->prof.live.push_back(rec);
        }
    }
};

// ------------------------------------------------------------------------------------------
// Debug build (python -m paper_2507_21684_b200.build --bounds, i.e. -DSPH_BOUNDS): every shared-memory gather index, ring
// offset and staging offset of the tile kernels is checked; a violation prints its source line and is counted in
// sph_bounds_count (read with sph_debug_bounds_violations()).  compute-sanitizer is closed on the GPU pool this was
// developed on; this stands in for memcheck on the hand-carved shared-memory layouts.
#ifdef SPH_BOUNDS
#include <stdio.h>
static __device__ unsigned int sph_bounds_count = 0;   // one per translation unit (no -rdc); summed by sph_api.cu
#define SPH_ASSERT(cond)                                                                                              \
    do {                                                                                                              \
        if (!(cond)) {                                                                                                \
            if (atomicAdd(&sph_bounds_count, 1u) < 16u)                                                               \
                printf("SPH_BOUNDS %s:%d block %d thread %d: %s\n", __FILE__, __LINE__, (int)blockIdx.x,              \
                       (int)threadIdx.x, #cond);                                                                      \
        }                                                                                                             \
    } while (0)
#else
#define SPH_ASSERT(cond) ((void)0)
#endif

// ------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float fast_sqrt(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));   // one MUFU.SQRT (no denormal fix-up code)
    return r;
}
__device__ __forceinline__ float fast_rcp(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));    // one MUFU.RCP
    return r;
}

// 10-bit-per-axis (3D) / 16-bit-per-axis (2D) Morton interleave
__device__ __forceinline__ uint32_t spread3(uint32_t v)
{
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__device__ __forceinline__ uint32_t compact3(uint32_t v)
{
    v &= 0x09249249u;
    v = (v | (v >> 2)) & 0x030c30c3u;
    v = (v | (v >> 4)) & 0x0300f00fu;
    v = (v | (v >> 8)) & 0x030000ffu;
    v = (v | (v >> 16)) & 0x3ffu;
    return v;
}
__device__ __forceinline__ uint32_t spread2(uint32_t v)
{
    v &= 0xffffu;
    v = (v | (v << 8)) & 0x00ff00ffu;
    v = (v | (v << 4)) & 0x0f0f0f0fu;
    v = (v | (v << 2)) & 0x33333333u;
    v = (v | (v << 1)) & 0x55555555u;
    return v;
}
__device__ __forceinline__ uint32_t compact2(uint32_t v)
{
    v &= 0x55555555u;
    v = (v | (v >> 1)) & 0x33333333u;
    v = (v | (v >> 2)) & 0x0f0f0f0fu;
    v = (v | (v >> 4)) & 0x00ff00ffu;
    v = (v | (v >> 8)) & 0xffffu;
    return v;
}
__device__ __forceinline__ uint32_t morton_encode(int dim, int cx, int cy, int cz)
{
    return dim == 3 ? (spread3(cx) | (spread3(cy) << 1) | (spread3(cz) << 2)) : (spread2(cx) | (spread2(cy) << 1));
}
__device__ __forceinline__ void morton_decode(int dim, uint32_t key, int &cx, int &cy, int &cz)
{
    if (dim == 3) {
        cx = (int)compact3(key);
        cy = (int)compact3(key >> 1);
        cz = (int)compact3(key >> 2);
    } else {
        cx = (int)compact2(key);
        cy = (int)compact2(key >> 1);
        cz = 0;
    }
}

// R4: binary32, every operation rounded separately, no contraction.
__device__ __forceinline__ float wrap_coord(float x, float lo, float hi, float L)
{
    float a = __fsub_rn(x, lo);
    float t = __fdiv_rn(a, L);
    float f = floorf(t);
    float p = __fmul_rn(L, f);
    float w = __fsub_rn(x, p);
    if (w >= hi) w = __fsub_rn(w, L);
    if (w < lo) w = __fadd_rn(w, L);
    return w;
}

// cell coordinate of a (possibly out-of-box) coordinate: monotone in x (binary64 sub, div, floor)
__device__ __forceinline__ int cell_coord_raw(double x, double lo, double edge)
{
    return (int)floor(__ddiv_rn(__dsub_rn(x, lo), edge));
}

// host-side launch helpers implemented in the .cu files
int sph_tile_expand_col(sph_ctx *ctx, cudaStream_t st);   // tile-local lists -> 32-bit sorted ids in ctx->col
int sph_launch_density_tile(sph_ctx *ctx, const KPar &kp, const float *m_s, float *rho_out, const uint32_t *um,
                            const float *m_caller, cudaStream_t st);
int sph_launch_density_vjp_tile(sph_ctx *ctx, const KPar &kp, const float2 *mr_s, float *x_bar, float *m_bar,
                                cudaStream_t st);
int sph_launch_grad_sum_tile(sph_ctx *ctx, const KPar &kp, const float *a_s, float *g_out, cudaStream_t st);
// the list build of sph_rk_step on its own (sph_step_host runs it before it queues its result copies: the small
// read-backs of the build would otherwise wait behind those copies in the device-to-host copy engine)
int sph_rk_prepare_lists(sph_ctx *ctx, const sph_domain *dom, float skin, const float *x, const float *h, int64_t n,
                         cudaStream_t st);
int sph_lists_valid_impl(sph_ctx *ctx, const float *x, const float *h, float skin_needed, int32_t *valid_out,
                         float *max_disp_out, cudaStream_t st);
int sph_launch_renorm_vjp_tile(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *rb, const float4 *rc,
                               const float2 *rd, const float *re, const uint32_t *perm, float *x_bar, float *vol_bar,
                               float *A_bar, cudaStream_t st);
int sph_launch_renorm_tile(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float2 *va_s, float4 *mom, cudaStream_t st);
int sph_launch_delta_term_tile(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *g4, const float2 *lr,
                               bool adjoint, float *drho_io, float4 *out4_io, float4 *dx4, float4 *gb4, float *partial,
                               cudaStream_t st);
// delta_form 1 (sph_delta.cu): the second part of the delta-term of [43] on top of a finished RHS / VJP launch
int sph_delta_forward(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2, float *drho,
                      float4 *out4, cudaStream_t st);
int sph_delta_adjoint(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2, const float4 *cot,
                      float *xb, float *rb, float4 *xb4, float *params_bar, cudaStream_t st);
// renormalisation passes on given sorted positions (sph_pairs.cu)
int sph_renorm_moments_any(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float2 *va_s, float4 *mom, cudaStream_t st);
int sph_renorm_vjp_pairs_any(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *rb, const float4 *rc,
                             const float2 *rd, const float *re, const uint32_t *perm, float *x_bar, float *vol_bar,
                             float *A_bar, cudaStream_t st);
int sph_delta_term_generic(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *g4, const float2 *lr, bool adjoint,
                           float *drho_io, float4 *out4_io, float4 *dx4, float4 *gb4, float *partial, int *npartial,
                           cudaStream_t st);
int sph_renorm_solve_sorted(sph_ctx *ctx, const KPar &kp, const float4 *mom, const float2 *va_s, const float4 *gbar4,
                            float4 *g4_out, float4 *rb, float4 *rc, float2 *rd, float *re, cudaStream_t st);
int sph_launch_grad_sum_vjp_tile(sph_ctx *ctx, const KPar &kp, const float4 *ga_s, float *x_bar, float *a_bar,
                                 cudaStream_t st);
int sph_launch_rhs_tile(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                        const uint8_t *kind_s, float *drho, float *acc, float4 *out4, cudaStream_t st);
int sph_vjp_tile_split(const sph_ctx *ctx, const KPar &kp);
int sph_launch_vjp_tile(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                        const float4 *cot, const float4 *eos, float *xb, float *vb, float *rb, float4 *xb4, float4 *vb4,
                        float *partials, cudaStream_t st);
struct SearchPar;
int sph_fused_stats_launch(sph_ctx *ctx, cudaStream_t st);
int sph_neighbors_fused_run(sph_ctx *ctx, const SearchPar &sp, const TileGeom &tg, uint32_t Mmax, uint32_t Tmax,
                            uint32_t ncmax, unsigned long long pairs_bound, cudaStream_t st, int64_t *nnz_out);
int sph_scan_u32(sph_ctx *ctx, const uint32_t *in, void *out, bool out64, int64_t m, cudaStream_t st);
int sph_kpar_make(const sph_ctx *ctx, const sph_params *par, KPar *kp);
int sph_launch_rhs_sorted(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                          const uint8_t *kind_s, float *drho, float *acc, float4 *out4, cudaStream_t st);
int sph_launch_vjp_sorted(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                          const float4 *cot, const float4 *eos, float *xb, float *vb, float *rb, float4 *xb4,
                          float4 *vb4, float *params_bar, int accumulate_params, cudaStream_t st);
