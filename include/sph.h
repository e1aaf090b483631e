/*
 * sph.h -- C ABI of the B200-native delta-SPH right-hand side and adjoint
 *          (data-parallel hot path of diffSPH, arXiv 2507.21684; text at PAPER.md).
 *
 * Conventions (apply to every call unless stated otherwise)
 *   - All array arguments are DEVICE pointers owned by the caller (e.g. PyTorch tensors), contiguous:
 *       x, v, acc, x_bar, v_bar, acc_bar : float [n][dim] row-major
 *       rho, m, h, drho_dt, ...          : float [n]
 *       kind                             : uint8 [n]   0 = fluid, 1 = fixed boundary particle
 *     "h" is the SUPPORT RADIUS H of the kernel ("we chose to denote the support itself as h").
 *   - Every call enqueues its work on `stream` and returns without synchronising, except
 *     sph_neighbors / sph_rk_step / sph_rk_step_vjp / sph_check (they read nnz / the error flag back) and
 *     the *_host convenience entry points.
 *   - The context owns sorted copies, keys, cell tables, the CSR and scratch (grown on demand).
 *     Outputs are always in the CALLER's particle order.
 *   - Return value: 0 = SPH_OK, negative = error code below.  No exceptions, no aborts, no printing.
 *   - There is no CPU fallback anywhere behind this interface.
 *
 * What is computed (readings R1..R9 are listed in DESIGN.md):
 *   Wendland C4 kernel  W = C_d/H^d (1-q)_+^6 (1+6q+35/3 q^2), C_2 = 9/pi, C_3 = 495/(32 pi)
 *   H_ij = max(h_i,h_j)  (BASELINE.json config 4),  smoothing scale l = H/kappa_d
 *   N(i) = { j : |x_i - x_j|^2 < (search_scale*H_ij)^2 } with minimum image on periodic axes, self included
 *   rho_i     = sum_j m_j W_ij                                                             PAPER.md:91 Eq.8
 *   drho_i/dt = sum_j [ rho_i V_j (v_i-v_j).grad_i W_ij  +  2 delta l c0 V_j (rho_i-rho_j) r^2/(r^2+(eps H)^2) G ]
 *                                                                     PAPER.md:95 Eq.9; Eq.42
 *   a_i       = sum_j [ -m_j (p_i/rho_i^2 + p_j/rho_j^2) + eta rho0 V_j (v_ij.x_ij)/(rho_i (r^2+(eps H)^2)) ] grad_i W_ij + g
 *               eta = alpha l c0 + 2(d+2) nu;   a_i = 0 for boundary kinds            PAPER.md:497 Eq.40; 87 Eq.7
 *   p         = rho0 c0^2/gamma ((rho/rho0)^gamma - 1)                                     PAPER.md:112 Eq.12
 *   with V_j = m_j/rho_j and grad_i W_ij = G (x_i - x_j).
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* opaque CUDA stream handle (binary compatible with cudaStream_t); NULL = the legacy default stream */
typedef struct CUstream_st *sph_stream_t;

typedef struct sph_ctx sph_ctx; /* opaque */

/* Simulation box and cell grid.  PAPER.md:556 (cells of size c), PAPER.md:165 (periodic via modulo). */
typedef struct {
    int dim;          /* 2 or 3 */
    int periodic[3];  /* per axis: 1 = periodic (positions wrapped into [lo,hi), minimum image), 0 = bounded */
    float lo[3];      /* lower corner; bounded axes: every position must lie in [lo,hi) */
    float hi[3];      /* upper corner */
    float cell_size;  /* >= largest search radius search_scale*max(h).  Periodic axes use the edge
                         L/floor(L/cell_size) (>= cell_size, at least 3 cells); bounded axes use cell_size. */
} sph_domain;

/* Global parameters ("global state dictionary C").  sph_rhs_vjp returns the gradient with
 * respect to the first ten floats in this order: c0, rho0, gamma, delta, alpha, nu, eps, g[0], g[1], g[2]. */
typedef struct {
    float c0;     /* speed of sound, > 0 */
    float rho0;   /* rest density, > 0 */
    float gamma;  /* Tait exponent (7) */
    float delta;  /* delta-SPH density diffusion coefficient PAPER.md:103 */
    float alpha;  /* artificial viscosity */
    float nu;     /* kinematic viscosity                     PAPER.md:83 Eq.6 */
    float eps;    /* regularisation of 1/r^2 relative to H, > 0 */
    float g[3];   /* body force (gravity) */
    int pressure_form; /* 0 = symmetric Eq.40: -m_j (p_i/rho_i^2 + p_j/rho_j^2);  1 = -m_j (p_i + p_j)/(rho_i rho_j), the form
                          the paper's own WCSPH scheme uses;  others: SPH_E_INVALID */
    int delta_form;    /* density diffusion (the equation is not printed, R6 / R17):
                          0 = Molteni-Colagrossi: delta l c0 sum_j 2 (rho_i - rho_j) r^2/(r^2 + (eps H)^2) G V_j;
                          1 = the delta-SPH term of Antuono et al. [43]: the same minus
                              delta l c0 sum_j V_j (g_i + g_j).(x_i - x_j) G  with g = <grad rho>^L, the renormalised density
                              gradient of PAPER.md:524-528 Eq.44/45 (zero diffusion of linear density fields up to the
                              free surface).  sph_rhs then runs the renormalisation passes first; sph_rhs_vjp
                              differentiates through L_i.  others: SPH_E_INVALID */
    float renorm_rcond; /* delta_form 1: eigenvalues of the renormalisation matrix below renorm_rcond * largest are dropped
                          in the pseudo-inverse; 0 <= renorm_rcond < 1, e.g. 1e-4 */
} sph_params;

enum {
    SPH_OK = 0,
    SPH_E_INVALID = -1, /* null pointer, n <= 0, dim not 2/3, eps <= 0, c0/rho0 <= 0, unsupported option */
    SPH_E_DOMAIN = -2,  /* cell_size < search radius, < 3 cells on a periodic axis, hi <= lo, too many cells,
                           non-finite or out-of-box position on a bounded axis, h or rho not a positive finite
                           number, non-finite mass (detected on device in a sticky flag that sph_build_cells
                           clears; reported by sph_neighbors, the *_host calls and sph_check) */
    SPH_E_STATE = -3,   /* call order violated (neighbours before cells, RHS before neighbours, different n) */
    SPH_E_NOMEM = -4,   /* device or host allocation failed */
    SPH_E_CUDA = -5,    /* a CUDA runtime call failed */
    SPH_E_TOO_LARGE = -6 /* size beyond the fixed capacity of an allocation-free entry point (sph_prefix_sum_noalloc) */
};

/* Create a context on CUDA device `device`.  n_max is a sizing hint (scratch grows on demand). */
int sph_create(sph_ctx **out, int device, int64_t n_max);
int sph_destroy(sph_ctx *ctx);

/* Steps N1-N4 of SURVEY.md 8(a): wrap positions, Morton cell key, stable radix sort,
 * reorder into sorted float4 SoA, cell start/end table.  x: [n][dim], h: [n].  Keeps n for later calls. */
int sph_build_cells(sph_ctx *ctx, const sph_domain *dom, const float *x, const float *h, int64_t n,
                    sph_stream_t stream);

/* Steps N5-N7 (count / exclusive scan / fill): compact CSR neighbour lists of the positions given
 * to sph_build_cells, radius search_scale*max(h_i,h_j), search_scale >= 1 (a Verlet skin).
 * Synchronises `stream`; *nnz_out (host pointer, may be NULL) receives the number of entries. */
int sph_neighbors(sph_ctx *ctx, float search_scale, int64_t *nnz_out, sph_stream_t stream);

/* Verlet-list validity ("the neighbor list needs to be updated if any particle
 * moves more than half of the skin-width ... with respect to the positions used during the original neighborhood
 * query"): D = max_i |x_i - x_build_i| (minimum image on periodic axes) of the positions x [n][dim] against those given
 * to sph_build_cells.  *valid_out = 1 iff 2 D <= (search_scale - 1 - skin_needed) * min h, i.e. every pair closer than
 * (1 + skin_needed) * H_ij at x is still in the lists of the last sph_neighbors(search_scale).  valid_out and
 * max_disp_out are HOST pointers (either may be NULL).  Synchronises `stream`. */
int sph_lists_valid(sph_ctx *ctx, const float *x, float skin_needed, int32_t *valid_out, float *max_disp_out,
                    sph_stream_t stream);

/* Copy the lists out in CALLER ids: row_ptr [n+1] int64, col_idx [nnz] int32, each row ascending, self included. */
int sph_neighbors_export(sph_ctx *ctx, int64_t *row_ptr, int32_t *col_idx, sph_stream_t stream);

/* rho_i = sum_{j in N(i)} m_j W(r_ij, max(h_i,h_j)) at the positions given to sph_build_cells.  PAPER.md:91 Eq.8 */
int sph_density(sph_ctx *ctx, const float *m, float *rho_out, sph_stream_t stream);

/* Reverse-mode adjoint of sph_density (the paper's backward benchmark differentiates the
 * summation density w.r.t. the positions; density-matching loss PAPER.md:353 Eq.21): given
 * rho_bar = dL/d rho [n], writes x_bar [n][dim] = sum_j (rho_bar_i m_j + rho_bar_j m_i) G_ij (x_i - x_j) and, if
 * m_bar is not NULL, m_bar [n] = sum_j rho_bar_j W_ij, at the positions given to sph_build_cells, adjacency fixed
 * (PAPER.md:161), h not differentiated.  Gather form over the symmetric lists: no atomics. */
int sph_density_vjp(sph_ctx *ctx, const float *m, const float *rho_bar, float *x_bar, float *m_bar,
                    sph_stream_t stream);

/* Kernel-gradient sum with per-particle weights (the gradient term of the particle-shifting loss,
 * PAPER.md:379 Eq.24, with a_j = m_j/rho_j): g_i = sum_j a_j grad_i W_ij = sum_j a_j G_ij (x_i - x_j), g_out [n][dim], at
 * the positions given to sph_build_cells. */
int sph_grad_sum(sph_ctx *ctx, const float *a, float *g_out, sph_stream_t stream);

/* Reverse-mode adjoint of sph_grad_sum with the exact kernel Hessian G Id + K d d^T: given
 * g_bar [n][dim], writes x_bar [n][dim] = sum_j [ a_j (G g_bar_i + K (d.g_bar_i) d) - a_i (G g_bar_j + K (d.g_bar_j) d) ]
 * and, if a_bar is not NULL, a_bar [n] = - sum_j G_ij (x_i - x_j) . g_bar_j.  Adjacency fixed; gather form, no atomics. */
int sph_grad_sum_vjp(sph_ctx *ctx, const float *a, const float *g_bar, float *x_bar, float *a_bar,
                     sph_stream_t stream);

/* Kernel renormalisation, Eq.44 and Eq.45, on the lists of the last sph_neighbors and at the build
 * positions: with V_j = vol[j] (the caller passes m_j/rho_j) and grad_i W_ij = G_ij (x_i - x_j),
 *     L_i = [ sum_j V_j (x_j - x_i) (x) grad_i W_ij ]^+                 (Eq.45; the matrix is symmetric)
 *     <grad A>_i = sum_j V_j (A_j - A_i) L_i grad_i W_ij                  (Eq.44)
 * ^+ is the Moore-Penrose inverse taken by eigen-decomposition: eigenvalues with |lambda| <= rcond * max|lambda| are
 * dropped ("commonly performed as a pseudo-inverse for numerical stability"), so a particle without
 * neighbours gets L = 0 and particles on a line / in a plane get the gradient within it.  0 <= rcond < 1.
 * vol, A: device float[n] in caller order.  L_out: device float[n*d*d], row-major d x d per particle, or NULL;
 * grad_out: device float[n*d] or NULL (not both NULL).  All buffers stay owned by the caller.  Returns SPH_E_INVALID on bad arguments, SPH_E_STATE without lists. */
int sph_renorm_gradient(sph_ctx *ctx, const float *vol, const float *A, float rcond, float *L_out, float *grad_out,
                        sph_stream_t stream);

/* Reverse-mode adjoint of the corrected gradient of sph_renorm_gradient ("fully supports backpropagation through this
 * operation as well"), adjacency held fixed: given grad_bar (device float[n*d], the cotangent
 * of <grad A>), writes x_bar (float[n*d]), vol_bar (float[n] or NULL) and A_bar (float[n] or NULL).  The moments are
 * recomputed (nothing is kept between calls); the pseudo-inverse is differentiated at constant rank
 * (d M^+ = -M^+ dM M^+ + (I - M M^+) dM M^+ M^+ on the range of the data), exact wherever no eigenvalue crosses the cutoff.
 * Gather form over the symmetric list, no atomics, bit-reproducible.  Same argument rules and errors as the forward. */
int sph_renorm_gradient_vjp(sph_ctx *ctx, const float *vol, const float *A, float rcond, const float *grad_bar,
                            float *x_bar, float *vol_bar, float *A_bar, sph_stream_t stream);

/* One right-hand-side evaluation (formulas at the top of this file) on the lists of the last sph_neighbors.
 * x may differ from the build positions (RK stages) as long as the list is still a superset of the true
 * neighbours: pairs with r >= H_ij contribute exactly 0 (kernel clamp).  h is the one given to sph_build_cells. */
int sph_rhs(sph_ctx *ctx, const sph_params *par, const float *x, const float *v, const float *rho,
            const float *m, const uint8_t *kind, float *drho_dt, float *acc, sph_stream_t stream);

/* Reverse-mode adjoint of sph_rhs (pair terms recomputed; adjacency fixed):
 * given drho_bar = dL/d(drho_dt) [n] and acc_bar = dL/d(acc) [n][dim], writes x_bar, v_bar [n][dim], rho_bar [n]
 * and params_bar[10] (DEVICE pointer; order as in sph_params; may be NULL). */
int sph_rhs_vjp(sph_ctx *ctx, const sph_params *par, const float *x, const float *v, const float *rho,
                const float *m, const uint8_t *kind, const float *drho_bar, const float *acc_bar,
                float *x_bar, float *v_bar, float *rho_bar, float *params_bar, sph_stream_t stream);

/* One classic RK4 step of y = (x, v, rho), f = (v, a, drho/dt); boundary kinds keep x and v.
 * Rebuilds cells and lists from x with search_scale = 1 + skin (skin >= 0; the caller guarantees
 * skin*min(h) >= 2*dt*max|v| so that one list serves the four stages).  x, v, rho: in/out. */
int sph_rk_step(sph_ctx *ctx, const sph_domain *dom, const sph_params *par, float dt, float skin, int64_t n,
                float *x, float *v, float *rho, const float *m, const float *h, const uint8_t *kind,
                sph_stream_t stream);

/* Discrete adjoint of sph_rk_step (stages recomputed from the step's initial state):
 * x0, v0, rho0_state = state at t; x_bar, v_bar, rho_bar hold dL/dy(t+dt) on entry and dL/dy(t) on return;
 * params_bar[10] (device, may be NULL) is ACCUMULATED into. */
int sph_rk_step_vjp(sph_ctx *ctx, const sph_domain *dom, const sph_params *par, float dt, float skin, int64_t n,
                    const float *x0, const float *v0, const float *rho0_state, const float *m, const float *h,
                    const uint8_t *kind, float *x_bar, float *v_bar, float *rho_bar, float *params_bar,
                    sph_stream_t stream);

/* Particle shifting at the end of a step (the scheme of [41] is not printed: reading R18 of DESIGN.md
 * takes the Fickian form along the gradient of the particle concentration):
 *     x_i <- x_i - theta l_i^2 sum_j (m_j/rho_j) grad_i W_ij     for fluid kinds (kind 0),  l_i = h_i / kappa_d,
 * evaluated at the CURRENT positions x on the lists of the last sph_neighbors / sph_rk_step (they must still be a
 * superset of the neighbours: e.g. directly after sph_rk_step, whose lists carry the skin).  x: in/out. */
int sph_shift(sph_ctx *ctx, float theta, float *x, const float *m, const float *rho, const uint8_t *kind,
              sph_stream_t stream);

/* End-to-end convenience call with HOST buffers (pageable or pinned): copies the inputs to the device, runs
 * sph_build_cells + sph_neighbors(search_scale) + sph_rhs + sph_rhs_vjp, copies the seven outputs back and
 * synchronises.  Output pointers may be NULL (skipped).  params_bar: host float[10]. */
int sph_forward_backward_host(sph_ctx *ctx, const sph_domain *dom, const sph_params *par, float search_scale,
                              int64_t n, const float *x, const float *v, const float *rho, const float *m,
                              const float *h, const uint8_t *kind, const float *drho_bar, const float *acc_bar,
                              float *drho_dt, float *acc, float *x_bar, float *v_bar, float *rho_bar,
                              float *params_bar, int64_t *nnz_out);

/* End-to-end call of ONE WHOLE STEP of the hot path with HOST buffers (all SURVEY.md 8(a) rows): copies the state and
 * the cotangents to the device, then sph_build_cells + sph_neighbors(1) + sph_density + sph_rhs + sph_rhs_vjp on the
 * grid of `dom`, then sph_rk_step(dt, skin) on the grid of `dom_rk` (cell_size >= (1+skin) max h), copies every result
 * back and synchronises.  x, v, rho are advanced IN PLACE (host); the other outputs may be NULL (skipped).
 * nnz_out[2] (host): entries of the two lists (exact radius; skin radius). */
int sph_step_host(sph_ctx *ctx, const sph_domain *dom, const sph_domain *dom_rk, const sph_params *par, float dt,
                  float skin, int64_t n, float *x, float *v, float *rho, const float *m, const float *h,
                  const uint8_t *kind, const float *drho_bar, const float *acc_bar, float *density, float *drho_dt,
                  float *acc, float *x_bar, float *v_bar, float *rho_bar, float *params_bar, int64_t *nnz_out);

/* Allocation-free exclusive prefix sum: step N6 of the neighbour build (per-row counts -> 64-bit CSR offsets,
 * PAPER.md:557-558 App. B step 2) for callers that cannot call cudaMalloc -- code under CUDA graph capture, tight
 * serving loops, harnesses that forbid allocation.  It needs no sph_ctx and calls no cudaMalloc / cudaFree / allocating
 * library routine: the block sums of the scan live in a fixed device array inside the library (128 KiB on every GPU
 * that loads it, until exit), which limits n to SPH_PREFIX_SUM_NOALLOC_MAX.
 *   device : CUDA device of the buffers; made current (and left current), as every other call does with its context's
 *   counts : device uint32[n], read only;   offsets: device int64[n + 1], written: offsets[i] = counts[0] + ... +
 *            counts[i-1], offsets[n] = the total.  Both stay owned by the caller; they must not overlap.
 *   n      : 0 <= n <= SPH_PREFIX_SUM_NOALLOC_MAX.  n == 0 does the per-device set-up only (one symbol look-up, no
 *            launch): call it once per device BEFORE a stream capture starts; later calls only launch three kernels on
 *            `stream`, asynchronously.
 * Returns SPH_E_TOO_LARGE for n beyond the maximum (nothing is launched), SPH_E_INVALID for a null pointer, negative n
 * or a device number outside 0..63, SPH_E_CUDA if the runtime fails.
 * All calls on a device share the one scratch array.  Its old contents never matter (every word a call reads it has
 * written first), but two calls whose kernels OVERLAP on the GPU -- different streams without an ordering between
 * them, or several host threads -- race on it and both results are garbage: order them on one stream or by events. */
#define SPH_PREFIX_SUM_NOALLOC_MAX (1ll << 26)
int sph_prefix_sum_noalloc(int device, const uint32_t *counts, int64_t *offsets, int64_t n, sph_stream_t stream);

/* Fetch the device-side error flag (synchronises the context's last stream). */
int sph_check(sph_ctx *ctx);
/* Debug builds only (python -m paper_2507_21684_b200.build --bounds, -DSPH_BOUNDS: every shared-memory gather index,
 * ring offset and staging offset of the tile kernels is a checked access).  *count (host) = violations seen since the
 * library was loaded (the first 16 also print their source line); -1 when the library is not a debug build.
 * Synchronises the device. */
int sph_debug_bounds_violations(sph_ctx *ctx, int64_t *count);
const char *sph_strerror(int code);

/* Introspection for tests / bench (host values of the last build): grid size per axis, nnz, number of kernels
 * launched by this context since creation. */
int sph_get_info(sph_ctx *ctx, int32_t ncell[3], int64_t *n, int64_t *nnz, int64_t *launches);

/* Layout of the lists built by the last sph_neighbors: *mode = 1 generic (32-bit sorted ids) or 2 tile-local (16-bit
 * indices into the halo of a block of tile_edge^dim cells); halo_max / rows_max = largest halo population / row count
 * of a block (0 for the generic layout).  Any pointer may be NULL. */
int sph_get_layout(sph_ctx *ctx, int32_t *mode, int32_t *tile_edge, int64_t *halo_max, int64_t *rows_max);

/* Per-kernel-class device timing for the roofline report (bench.py): when enabled, every launch (group) of a class
 * is bracketed by two CUDA events on the launching stream.  sph_profile_read synchronises the device, adds the
 * resolved durations to ms_sum[SPH_K_NCLASS] (milliseconds) and the launch counts to launches[SPH_K_NCLASS]
 * (both host arrays, may be NULL), then clears the accumulators.  Classes follow SURVEY.md 8(a). */
enum {
    SPH_K_KEY = 0,   /* N1 wrap + cell key */
    SPH_K_SORT,      /* N2 radix passes (histogram, scan, scatter) */
    SPH_K_REORDER,   /* N3 + N4 sorted SoA, cell ranges */
    SPH_K_COUNT,     /* N5 */
    SPH_K_SCAN,      /* N6 */
    SPH_K_FILL,      /* N7 */
    SPH_K_EXPORT,    /* lists in caller ids */
    SPH_K_DENSITY,   /* D */
    SPH_K_PACK,      /* R0 gather into sorted SoA + EOS prologue, cotangent pack */
    SPH_K_RHS,       /* R1 pair loop */
    SPH_K_VJP,       /* B1 pair loop */
    SPH_K_REDUCE,    /* B2 */
    SPH_K_RK,        /* T stage updates (axpy) and adjoint bookkeeping */
    SPH_K_NCLASS
};
/* Tuning knobs (results do not depend on them beyond summation order). */
enum {
    SPH_OPT_PAIR_GROUP = 1, /* lanes that share one row in the pair kernels: 4, 8, 16, 32; 0 = default */
    SPH_OPT_LIST_MODE = 2,  /* internal list layout chosen by the next sph_neighbors: 0 = automatic; 1 = generic
                               (32-bit sorted ids, neighbour state gathered through L1/L2, any cell occupancy);
                               2 = tile-local (16-bit indices into the halo of a block of cells, neighbour state staged
                               in shared memory).  2 falls back to 1 when a halo does not fit shared memory. */
    SPH_OPT_TILE_EDGE = 3,  /* edge of the cell blocks of the tile-local layout: 1, 2, 4 cells; 0 = automatic */
    SPH_OPT_PAIR_WARPS = 4, /* warps per CTA of the tile pair kernels: 4, 8, 10, 12, 16, 20, 24 (capped by a kernel's launch
                               bound); 0 = automatic: the most resident warps shared memory and registers admit */
    SPH_OPT_FILL_MASKS = 5, /* 1 (default): the fill of the tile-local lists expands the hit masks saved by the count pass;
                               0: it repeats the distance tests (no mask buffer) */
    SPH_OPT_BUILD_FUSED = 8, /* 1 (default): the tile-local lists are built by ONE kernel per build (tests, offsets by a
                               decoupled look-back over the tiles, fill; the hit masks stay in shared memory);
                               0: count / scan / fill as three steps with the masks in global memory */
    SPH_OPT_UNIFORM_MASS_PATH = 7, /* 1 (default): in 3D with uniform h the tile pair kernels (sph_rhs, sph_rhs_vjp) are
                               enqueued in two variants -- one that assumes all masses equal and gathers 32 / 48
                               instead of 40 / 56 bytes per pair, one general -- and a device flag written by this
                               call's own pack kernel decides which of them runs (no host synchronisation);
                               sph_density does the same with a flag of its own (written by its mass gather): the
                               uniform-mass variant neither stages nor gathers the masses.
                               0: only the general variants are launched */
    SPH_OPT_STAGE_BULK = 9, /* 0 (default): the tile pair kernels stage a halo with one 16-byte cp.async per particle and
                               array; 1: sph_rhs / sph_rhs_vjp stage their float4 arrays with one cp.async.bulk per halo
                               cell and array, completing on one mbarrier per CTA (A/B measurement) */
    SPH_OPT_VJP_SPLIT = 10, /* 1 (default): in 3D on 2x2x2-cell tiles the adjoint pair kernel of sph_rhs_vjp gives each CTA HALF
                               a tile (one z-layer of its cells, staging the three layers of halo cells around it), so
                               that two CTAs are resident per SM and one stages while the other computes;
                               0: one CTA per tile (A/B measurement).  (The same split of the forward kernel was
                               measured slower and is not built in: profiles/r02_h.) */
    SPH_OPT_TILE_TABLES = 11, /* 1 (default): the per-tile tables (halo cell offsets, row ranges, periodic shifts) are computed
                               once per neighbour build and loaded by every tile kernel;  0: every CTA derives them from
                               the cell table again (A/B measurement) */
    SPH_OPT_RK_EXTRA_SKIN = 6 /* Verlet lists across steps: value/1000 = extra skin e (in units of h).  With
                               e > 0 sph_rk_step / sph_rk_step_vjp build their lists with search_scale = 1 + skin + e
                               (the domain's cell_size must cover it) and a later call with the same domain, n and h
                               REUSES them while sph_lists_valid(x, skin) holds (and h is unchanged: checked);
                               0: rebuilt in every call; -1 (default): automatic -- in 2D the lists take whatever the
                               domain's cell_size leaves above 1 + skin (at most 0.25) and are reused likewise, so a
                               caller opts in by passing larger cells; none in 3D, where it was measured not to pay */
};
int sph_set_option(sph_ctx *ctx, int key, int value);
int sph_profile_enable(sph_ctx *ctx, int on);
int sph_profile_read(sph_ctx *ctx, double *ms_sum, int64_t *launches);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
