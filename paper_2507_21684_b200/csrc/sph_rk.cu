// sph_rk.cu -- step T of SURVEY.md 8(a): classic RK4 of y = (x, v, rho),
// f(y) = (v, a, drho/dt), and its discrete adjoint with recomputed stages.
// All stage states live in the SORTED layout, so the four RHS evaluations run back to back on the pair
// kernels without permuting; one list with a Verlet skin serves the four stages.
#include "sph_internal.cuh"

#include <math.h>

namespace {

struct StageBufs {
    float4 *s0, *s1;
    float2 *s2;
    float4 *eos;
};

// Tait EOS prologue (same arithmetic as k_pack_state in sph_pairs.cu, kept local to this file)
__device__ __forceinline__ void eos_eval(const KPar &kp, float r, float mi, float &V, float &P, float4 *eos_out)
{
    const float u = (r - kp.rho0) / kp.rho0;
    const float lg = log1pf(u);
    const float ugm1 = expm1f(kp.gamma * lg);
    const float ug = ugm1 + 1.0f;
    const float pr = kp.Bp * ugm1;
    const float ir = 1.0f / r, ir2 = ir * ir;
    V = mi * ir;
    P = pr * ir2;
    if (eos_out) {
        const float dp_drho = kp.c0 * kp.c0 * ug / (1.0f + u);
        const float dP = dp_drho * ir2 - 2.0f * pr * ir2 * ir;
        const float dp_drho0 = kp.c0 * kp.c0 / kp.gamma * ugm1 - kp.c0 * kp.c0 * ug;
        const float dp_dgam = -kp.Bp / kp.gamma * ugm1 + kp.Bp * ug * lg;
        *eos_out = make_float4(dP, dp_drho0 * ir2, dp_dgam * ir2, mi);
    }
}

template <int DIM>
__device__ __forceinline__ void store_stage(const StageBufs &sb, int64_t p, const KPar &kp, const float *X,
                                            const float *Vv, float r, float mi, float h)
{
    float V, P;
    float4 e;
    eos_eval(kp, r, mi, V, P, sb.eos ? &e : nullptr);
    if (DIM == 3) {
        sb.s0[p] = make_float4(X[0], X[1], X[2], r);
        sb.s1[p] = make_float4(Vv[0], Vv[1], Vv[2], P);
        sb.s2[p] = make_float2(V, h);
    } else {
        sb.s0[p] = make_float4(X[0], X[1], Vv[0], Vv[1]);
        sb.s1[p] = make_float4(r, V, P, h);
    }
    if (sb.eos) sb.eos[p] = e;
}

// base state in sorted order: b0 = {xw,yw,zw,h}, b1 = {vx,vy,vz,rho}, m_s, kind_s; also writes stage 1 (= base)
template <int DIM>
__global__ void k_rk_base(int64_t n, KPar kp, const uint32_t *__restrict__ perm, const float4 *__restrict__ pos_s,
                          const float *__restrict__ x, const float *__restrict__ v, const float *__restrict__ rho,
                          const float *__restrict__ m,
                          const uint8_t *__restrict__ kind, float4 *__restrict__ b0, float4 *__restrict__ b1,
                          float *__restrict__ m_s, uint8_t *__restrict__ kind_s, StageBufs sb, uint32_t *__restrict__ um)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    const float m_first = __ldg(m);                          // uniform-mass flag pair (sph_um_flag)
    if (p == 0) um[1] = __float_as_uint(m_first);
    const float4 ps = pos_s[p];                              // wrapped build positions (R4) + h
    // current position: the periodic image next to the build position (identical to it when the lists were built
    // from x in this call; differs when Verlet lists are reused across steps)
    const float xb[3] = {ps.x, ps.y, ps.z};
    float X[3] = {0.f, 0.f, 0.f}, Vv[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        float xv = x[i * DIM + k];
        if (kp.periodic[k]) {
            xv = wrap_coord(xv, kp.lo[k], kp.hi[k], kp.L[k]);
            const float dd = xv - xb[k];
            xv = dd > kp.halfL[k] ? xv - kp.L[k] : (dd < -kp.halfL[k] ? xv + kp.L[k] : xv);
        }
        X[k] = xv;
        Vv[k] = v[i * DIM + k];
    }
    const float r = rho[i], mi = m[i];
    if (mi != m_first) um[0] = 0u;
    sph_flag_bad_state(um, r, mi);
    b0[p] = make_float4(X[0], X[1], X[2], ps.w);
    b1[p] = make_float4(Vv[0], Vv[1], Vv[2], r);
    m_s[p] = mi;
    kind_s[p] = kind[i];
    store_stage<DIM>(sb, p, kp, X, Vv, r, mi, ps.w);
}

// Y_s = y + c dt k_{s-1};  k_{s-1} = (v_{s-1} or 0 for boundary, a_{s-1}, drho_{s-1});  acc += b_{s-1} k_{s-1}
template <int DIM>
__global__ void k_rk_stage(int64_t n, KPar kp, float cdt, float bprev, int first, const float4 *__restrict__ b0,
                           const float4 *__restrict__ b1, const float *__restrict__ m_s,
                           const uint8_t *__restrict__ kind_s, const float4 *__restrict__ k4,
                           StageBufs prev, StageBufs sb, float4 *__restrict__ accx, float4 *__restrict__ accv)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float4 k = k4[p];                                  // {a, drho} of the previous stage
    float vp[3];
    if (DIM == 3) { const float4 t = prev.s1[p]; vp[0] = t.x; vp[1] = t.y; vp[2] = t.z; }
    else { const float4 t = prev.s0[p]; vp[0] = t.z; vp[1] = t.w; vp[2] = 0.f; }
    const bool fixed = kind_s[p] != 0;
    if (fixed) vp[0] = vp[1] = vp[2] = 0.f;                  // dx/dt = 0 for boundary kinds
    float4 ax = first ? make_float4(0.f, 0.f, 0.f, 0.f) : accx[p];
    float4 av = first ? make_float4(0.f, 0.f, 0.f, 0.f) : accv[p];
    ax.x = fmaf(bprev, vp[0], ax.x); ax.y = fmaf(bprev, vp[1], ax.y); ax.z = fmaf(bprev, vp[2], ax.z);
    ax.w = fmaf(bprev, k.w, ax.w);
    av.x = fmaf(bprev, k.x, av.x); av.y = fmaf(bprev, k.y, av.y); av.z = fmaf(bprev, k.z, av.z);
    accx[p] = ax;
    accv[p] = av;
    const float4 x0 = b0[p], v0 = b1[p];
    float X[3] = {fmaf(cdt, vp[0], x0.x), fmaf(cdt, vp[1], x0.y), fmaf(cdt, vp[2], x0.z)};
    float Vv[3] = {fmaf(cdt, k.x, v0.x), fmaf(cdt, k.y, v0.y), fmaf(cdt, k.z, v0.z)};
    const float r = fmaf(cdt, k.w, v0.w);
    store_stage<DIM>(sb, p, kp, X, Vv, r, m_s[p], x0.w);
}

// y(t+dt) = y + dt (acc + b_4 k_4), written to the caller's arrays in place (absolute positions are kept,
// only the increment is added to the unwrapped x)
template <int DIM>
__global__ void k_rk_final(int64_t n, float dt, float blast, const uint32_t *__restrict__ perm,
                           const uint8_t *__restrict__ kind_s, const float4 *__restrict__ k4, StageBufs last,
                           const float4 *__restrict__ accx, const float4 *__restrict__ accv, float *__restrict__ x,
                           float *__restrict__ v, float *__restrict__ rho)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    const float4 k = k4[p];
    float vp[3];
    if (DIM == 3) { const float4 t = last.s1[p]; vp[0] = t.x; vp[1] = t.y; vp[2] = t.z; }
    else { const float4 t = last.s0[p]; vp[0] = t.z; vp[1] = t.w; vp[2] = 0.f; }
    if (kind_s[p]) vp[0] = vp[1] = vp[2] = 0.f;
    const float4 ax = accx[p], av = accv[p];
    const float dx[3] = {fmaf(blast, vp[0], ax.x), fmaf(blast, vp[1], ax.y), fmaf(blast, vp[2], ax.z)};
    const float dv[3] = {fmaf(blast, k.x, av.x), fmaf(blast, k.y, av.y), fmaf(blast, k.z, av.z)};
#pragma unroll
    for (int kk = 0; kk < DIM; ++kk) {
        x[i * DIM + kk] = fmaf(dt, dx[kk], x[i * DIM + kk]);
        v[i * DIM + kk] = fmaf(dt, dv[kk], v[i * DIM + kk]);
    }
    rho[i] = fmaf(dt, fmaf(blast, k.w, ax.w), rho[i]);
}

// the same update for the caller indices [i0, i1) (one thread per caller index, gathers through inv_perm).
// WHAT: 1 = positions only, 2 = velocities and densities only, 3 = all.  The new positions need the velocities of the
// LAST stage state, not the last right-hand side, so sph_step_host has them computed (and copied out) while the fourth
// right-hand side still runs.
template <int DIM, int WHAT>
__global__ void k_rk_final_range(int64_t i0, int64_t i1, float dt, float blast, const uint32_t *__restrict__ inv_perm,
                                 const uint8_t *__restrict__ kind_s, const float4 *__restrict__ k4, StageBufs last,
                                 const float4 *__restrict__ accx, const float4 *__restrict__ accv, float *__restrict__ x,
                                 float *__restrict__ v, float *__restrict__ rho)
{
    const int64_t i = i0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= i1) return;
    const int64_t p = inv_perm[i];
    const float4 ax = accx[p];
    if (WHAT & 1) {
        float vp[3];
        if (DIM == 3) { const float4 t = last.s1[p]; vp[0] = t.x; vp[1] = t.y; vp[2] = t.z; }
        else { const float4 t = last.s0[p]; vp[0] = t.z; vp[1] = t.w; vp[2] = 0.f; }
        if (kind_s[p]) vp[0] = vp[1] = vp[2] = 0.f;
        const float dx[3] = {fmaf(blast, vp[0], ax.x), fmaf(blast, vp[1], ax.y), fmaf(blast, vp[2], ax.z)};
#pragma unroll
        for (int kk = 0; kk < DIM; ++kk) x[i * DIM + kk] = fmaf(dt, dx[kk], x[i * DIM + kk]);
    }
    if (WHAT & 2) {
        const float4 k = k4[p];
        const float4 av = accv[p];
        const float dv[3] = {fmaf(blast, k.x, av.x), fmaf(blast, k.y, av.y), fmaf(blast, k.z, av.z)};
#pragma unroll
        for (int kk = 0; kk < DIM; ++kk) v[i * DIM + kk] = fmaf(dt, dv[kk], v[i * DIM + kk]);
        rho[i] = fmaf(dt, fmaf(blast, k.w, ax.w), rho[i]);
    }
}

// ---- adjoint helpers ---------------------------------------------------------------------------------
// gather the incoming cotangents ybar(t+dt) into sorted order: yx = {xbar, rhobar}, yv = {vbar, 0}
template <int DIM>
__global__ void k_adj_gather(int64_t n, const uint32_t *__restrict__ perm, const float *__restrict__ xb,
                             const float *__restrict__ vb, const float *__restrict__ rb, float4 *__restrict__ yx,
                             float4 *__restrict__ yv)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    yx[p] = make_float4(xb[i * DIM], xb[i * DIM + 1], DIM == 3 ? xb[i * DIM + 2] : 0.f, rb[i]);
    yv[p] = make_float4(vb[i * DIM], vb[i * DIM + 1], DIM == 3 ? vb[i * DIM + 2] : 0.f, 0.f);
}

// kbar_s = b_s dt ybar+ + a_{s+1,s} dt Ybar_{s+1};  cot = {lambda = kbar_rho, mu = kbar_v (0 for boundary)};
// kbx = kbar_x (needed after the pair kernel: dx/dt = v  =>  vbar += kbar_x for fluid kinds)
__global__ void k_adj_cot(int64_t n, float bdt, float adt, const uint8_t *__restrict__ kind_s,
                          const float4 *__restrict__ yx, const float4 *__restrict__ yv, const float4 *__restrict__ Yx,
                          const float4 *__restrict__ Yv, float4 *__restrict__ cot, float4 *__restrict__ kbx)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float4 a = yx[p], b = yv[p];
    float4 kx = make_float4(bdt * a.x, bdt * a.y, bdt * a.z, bdt * a.w);   // {kbar_x, kbar_rho}
    float4 kv = make_float4(bdt * b.x, bdt * b.y, bdt * b.z, 0.f);
    if (adt != 0.f) {
        const float4 c = Yx[p], d = Yv[p];
        kx.x = fmaf(adt, c.x, kx.x); kx.y = fmaf(adt, c.y, kx.y); kx.z = fmaf(adt, c.z, kx.z); kx.w = fmaf(adt, c.w, kx.w);
        kv.x = fmaf(adt, d.x, kv.x); kv.y = fmaf(adt, d.y, kv.y); kv.z = fmaf(adt, d.z, kv.z);
    }
    const bool fixed = kind_s[p] != 0;
    cot[p] = fixed ? make_float4(kx.w, 0.f, 0.f, 0.f) : make_float4(kx.w, kv.x, kv.y, kv.z);
    kbx[p] = fixed ? make_float4(0.f, 0.f, 0.f, 0.f) : make_float4(kx.x, kx.y, kx.z, 0.f);
}

// Ybar_s.v += kbar_x ;  sum += Ybar_s
__global__ void k_adj_fix(int64_t n, int first, const float4 *__restrict__ kbx, const float4 *__restrict__ Yx,
                          float4 *__restrict__ Yv, float4 *__restrict__ sumx, float4 *__restrict__ sumv)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float4 k = kbx[p], a = Yx[p];
    float4 b = Yv[p];
    b.x += k.x; b.y += k.y; b.z += k.z;
    Yv[p] = b;
    float4 sx = first ? make_float4(0.f, 0.f, 0.f, 0.f) : sumx[p];
    float4 sv = first ? make_float4(0.f, 0.f, 0.f, 0.f) : sumv[p];
    sx.x += a.x; sx.y += a.y; sx.z += a.z; sx.w += a.w;
    sv.x += b.x; sv.y += b.y; sv.z += b.z;
    sumx[p] = sx;
    sumv[p] = sv;
}

// ybar(t) = ybar(t+dt) + sum_s Ybar_s, written back to the caller's arrays
template <int DIM>
__global__ void k_adj_final(int64_t n, const uint32_t *__restrict__ perm, const float4 *__restrict__ sumx,
                            const float4 *__restrict__ sumv, float *__restrict__ xb, float *__restrict__ vb,
                            float *__restrict__ rb)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    const float4 a = sumx[p], b = sumv[p];
    const float ax[3] = {a.x, a.y, a.z}, bv[3] = {b.x, b.y, b.z};
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        xb[i * DIM + k] += ax[k];
        vb[i * DIM + k] += bv[k];
    }
    rb[i] += a.w;
}

inline unsigned nb(int64_t n) { return (unsigned)((n + 255) / 256); }

// Lists for one step: cells and lists from x with search_scale = 1 + skin + e.  With an extra skin e > 0 the lists are kept
// across steps while no particle has moved more than half of it and h is unchanged.  e is
// SPH_OPT_RK_EXTRA_SKIN, or by default automatic: in 2D whatever the caller's cell size leaves above 1 + skin (capped at
// kAutoSkinCap; measured: 0.48 -> 0.29 ms per step at config 1, 1.35 -> 0.81 ms at config 2), none in 3D, where the
// longer lists cost more than the rebuilds saved (profiles/r01_d_final.md).
constexpr float kAutoSkinCap = 0.25f;
int rebuild(sph_ctx *ctx, const sph_domain *dom, float skin, const float *x, const float *h, int64_t n, cudaStream_t st)
{
    const bool automatic = ctx->opt_rk_extra_permille < 0;
    const float extra = automatic ? 0.f : 0.001f * (float)ctx->opt_rk_extra_permille;
    const bool reuse = automatic ? dom->dim == 2 : extra > 0.f;
    if (reuse && ctx->lists_ready && ctx->n == n && memcmp(&ctx->dom_last, dom, sizeof(*dom)) == 0 &&
        ctx->search_scale > 1.0f + skin) {
        int32_t ok = 0;
        SPH_TRY(sph_lists_valid_impl(ctx, x, h, skin, &ok, nullptr, st));
        if (ok) return SPH_OK;
    }
    SPH_TRY(sph_build_cells(ctx, dom, x, h, n, (sph_stream_t)st));
    if (automatic && dom->dim == 2) {
        ctx->scale_slack_cap = kAutoSkinCap;
        const int rc = sph_neighbors(ctx, 1.0f + skin, nullptr, (sph_stream_t)st);
        ctx->scale_slack_cap = 0.f;
        return rc;
    }
    return sph_neighbors(ctx, 1.0f + skin + extra, nullptr, (sph_stream_t)st);
}

} // namespace

int sph_rk_prepare_lists(sph_ctx *ctx, const sph_domain *dom, float skin, const float *x, const float *h, int64_t n,
                         cudaStream_t st)
{
    SPH_TRY(rebuild(ctx, dom, skin, x, h, n, st));
    ctx->rk_lists_prepared = true;
    return SPH_OK;
}

extern "C" int sph_rk_step(sph_ctx *ctx, const sph_domain *dom, const sph_params *par, float dt, float skin, int64_t n,
                           float *x, float *v, float *rho, const float *m, const float *h, const uint8_t *kind,
                           sph_stream_t stream)
{
    if (!ctx) return SPH_E_INVALID;
    const bool prepared = ctx->rk_lists_prepared;                    // built by sph_rk_prepare_lists for this call
    ctx->rk_lists_prepared = false;
    if (!dom || !par || !x || !v || !rho || !m || !h || !kind || !(skin >= 0.f)) return SPH_E_INVALID;
    if (n <= 0) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    if (!prepared || !ctx->lists_ready || ctx->n != n) SPH_TRY(rebuild(ctx, dom, skin, x, h, n, st));
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, par, &kp));
    SPH_TRY(ctx->s0.reserve((size_t)n * 16));
    SPH_TRY(ctx->s1.reserve((size_t)n * 16));
    SPH_TRY(ctx->s2.reserve((size_t)n * 8));
    SPH_TRY(ctx->kind_s.reserve((size_t)n));
    SPH_TRY(ctx->m_s.reserve((size_t)n * 4));
    SPH_TRY(ctx->out4.reserve((size_t)n * 16));
    for (int k = 0; k < 4; ++k) SPH_TRY(ctx->rk[k].reserve((size_t)n * 16));
    float4 *b0 = ctx->rk[0].as<float4>(), *b1 = ctx->rk[1].as<float4>();
    float4 *accx = ctx->rk[2].as<float4>(), *accv = ctx->rk[3].as<float4>();
    StageBufs sb{ctx->s0.as<float4>(), ctx->s1.as<float4>(), ctx->s2.as<float2>(), nullptr};
    float4 *k4 = ctx->out4.as<float4>();
    const uint32_t *perm = ctx->perm.as<uint32_t>();
    uint8_t *kind_s = ctx->kind_s.as<uint8_t>();
    float *m_s = ctx->m_s.as<float>();

    {
    KScope ks(ctx, SPH_K_RK, 1, st);
    SPH_CUDA_TRY(cudaMemsetAsync(sph_um_flag(ctx), 1, 4, st));
    if (kp.dim == 3)
        k_rk_base<3><<<nb(n), 256, 0, st>>>(n, kp, perm, ctx->pos_s.as<float4>(), x, v, rho, m, kind, b0, b1, m_s, kind_s, sb, sph_um_flag(ctx));
    else
        k_rk_base<2><<<nb(n), 256, 0, st>>>(n, kp, perm, ctx->pos_s.as<float4>(), x, v, rho, m, kind, b0, b1, m_s, kind_s, sb, sph_um_flag(ctx));
    }
    const float c[4] = {0.f, 0.5f, 0.5f, 1.f};
    const float b[4] = {1.f / 6.f, 1.f / 3.f, 1.f / 3.f, 1.f / 6.f};
    for (int s = 0; s < 4; ++s) {
        if (s > 0) {
            KScope ks(ctx, SPH_K_RK, 1, st);
            if (kp.dim == 3)
                k_rk_stage<3><<<nb(n), 256, 0, st>>>(n, kp, c[s] * dt, b[s - 1], s == 1, b0, b1, m_s, kind_s, k4, sb, sb, accx, accv);
            else
                k_rk_stage<2><<<nb(n), 256, 0, st>>>(n, kp, c[s] * dt, b[s - 1], s == 1, b0, b1, m_s, kind_s, k4, sb, sb, accx, accv);
        }
        if (s == 3 && ctx->rk_final_chunks > 1) {
            // sph_step_host: the new positions are complete before the last right-hand side (they need v of this stage
            // state only); the caller copies them out while it runs
            KScope ks(ctx, SPH_K_RK, 1, st);
            const uint32_t *inv_perm = ctx->inv_perm.as<uint32_t>();
            if (kp.dim == 3)
                k_rk_final_range<3, 1><<<nb(n), 256, 0, st>>>(0, n, dt, b[3], inv_perm, kind_s, k4, sb, accx, accv, x, v, rho);
            else
                k_rk_final_range<2, 1><<<nb(n), 256, 0, st>>>(0, n, dt, b[3], inv_perm, kind_s, k4, sb, accx, accv, x, v, rho);
            SPH_CUDA_TRY(cudaEventRecord(ctx->ev_final_x, st));
        }
        SPH_TRY(sph_launch_rhs_sorted(ctx, kp, sb.s0, sb.s1, sb.s2, kind_s, nullptr, nullptr, k4, st));
    }
    if (ctx->rk_final_chunks > 1) {
        // sph_step_host: ranges of caller indices, an event after each (the caller copies the range out meanwhile)
        const int C = ctx->rk_final_chunks;
        const uint32_t *inv_perm = ctx->inv_perm.as<uint32_t>();
        for (int cI = 0; cI < C; ++cI) {
            const int64_t i0 = n * cI / C, i1 = n * (cI + 1) / C;
            if (i1 > i0) {
                KScope ks(ctx, SPH_K_RK, 1, st);
                if (kp.dim == 3)
                    k_rk_final_range<3, 2><<<nb(i1 - i0), 256, 0, st>>>(i0, i1, dt, b[3], inv_perm, kind_s, k4, sb, accx, accv, x, v, rho);
                else
                    k_rk_final_range<2, 2><<<nb(i1 - i0), 256, 0, st>>>(i0, i1, dt, b[3], inv_perm, kind_s, k4, sb, accx, accv, x, v, rho);
            }
            SPH_CUDA_TRY(cudaEventRecord(ctx->ev_final[cI], st));
        }
    } else {
    KScope ks(ctx, SPH_K_RK, 1, st);
    if (kp.dim == 3)
        k_rk_final<3><<<nb(n), 256, 0, st>>>(n, dt, b[3], perm, kind_s, k4, sb, accx, accv, x, v, rho);
    else
        k_rk_final<2><<<nb(n), 256, 0, st>>>(n, dt, b[3], perm, kind_s, k4, sb, accx, accv, x, v, rho);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_rk_step_vjp(sph_ctx *ctx, const sph_domain *dom, const sph_params *par, float dt, float skin,
                               int64_t n, const float *x0, const float *v0, const float *rho0_state, const float *m,
                               const float *h, const uint8_t *kind, float *x_bar, float *v_bar, float *rho_bar,
                               float *params_bar, sph_stream_t stream)
{
    if (!ctx || !dom || !par || !x0 || !v0 || !rho0_state || !m || !h || !kind || !x_bar || !v_bar || !rho_bar ||
        !(skin >= 0.f))
        return SPH_E_INVALID;
    if (n <= 0) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    SPH_TRY(rebuild(ctx, dom, skin, x0, h, n, st));
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, par, &kp));
    // buffers: base (2), four stored stages (4 x {s0,s1,s2,eos}), k4, cotangent work arrays
    SPH_TRY(ctx->kind_s.reserve((size_t)n));
    SPH_TRY(ctx->m_s.reserve((size_t)n * 4));
    SPH_TRY(ctx->out4.reserve((size_t)n * 16));
    SPH_TRY(ctx->c0buf.reserve((size_t)n * 16));
    SPH_TRY(ctx->s0.reserve((size_t)n * 16 * 4));
    SPH_TRY(ctx->s1.reserve((size_t)n * 16 * 4));
    SPH_TRY(ctx->s2.reserve((size_t)n * 8 * 4));
    SPH_TRY(ctx->eos.reserve((size_t)n * 16 * 4));
    for (int k = 0; k < 12; ++k) SPH_TRY(ctx->rk[k].reserve((size_t)n * 16));
    float4 *b0 = ctx->rk[0].as<float4>(), *b1 = ctx->rk[1].as<float4>();
    float4 *accx = ctx->rk[2].as<float4>(), *accv = ctx->rk[3].as<float4>();
    float4 *yx = ctx->rk[4].as<float4>(), *yv = ctx->rk[5].as<float4>();
    float4 *Yx = ctx->rk[6].as<float4>(), *Yv = ctx->rk[7].as<float4>();
    float4 *sumx = ctx->rk[8].as<float4>(), *sumv = ctx->rk[9].as<float4>();
    float4 *kbx = ctx->rk[10].as<float4>();
    float4 *cot = ctx->c0buf.as<float4>();
    float4 *k4 = ctx->out4.as<float4>();
    StageBufs S[4];
    for (int s = 0; s < 4; ++s)
        S[s] = StageBufs{ctx->s0.as<float4>() + (size_t)s * n, ctx->s1.as<float4>() + (size_t)s * n,
                         ctx->s2.as<float2>() + (size_t)s * n, ctx->eos.as<float4>() + (size_t)s * n};
    const uint32_t *perm = ctx->perm.as<uint32_t>();
    uint8_t *kind_s = ctx->kind_s.as<uint8_t>();
    float *m_s = ctx->m_s.as<float>();
    const float c[4] = {0.f, 0.5f, 0.5f, 1.f};
    const float b[4] = {1.f / 6.f, 1.f / 3.f, 1.f / 3.f, 1.f / 6.f};

    // forward sweep: recompute and keep the four stage states
    {
    KScope ks(ctx, SPH_K_RK, 1, st);
    SPH_CUDA_TRY(cudaMemsetAsync(sph_um_flag(ctx), 1, 4, st));
    if (kp.dim == 3)
        k_rk_base<3><<<nb(n), 256, 0, st>>>(n, kp, perm, ctx->pos_s.as<float4>(), x0, v0, rho0_state, m, kind, b0, b1, m_s, kind_s, S[0], sph_um_flag(ctx));
    else
        k_rk_base<2><<<nb(n), 256, 0, st>>>(n, kp, perm, ctx->pos_s.as<float4>(), x0, v0, rho0_state, m, kind, b0, b1, m_s, kind_s, S[0], sph_um_flag(ctx));
    }
    for (int s = 1; s < 4; ++s) {
        SPH_TRY(sph_launch_rhs_sorted(ctx, kp, S[s - 1].s0, S[s - 1].s1, S[s - 1].s2, kind_s, nullptr, nullptr, k4, st));
        {
        KScope ks(ctx, SPH_K_RK, 1, st);
        if (kp.dim == 3)
            k_rk_stage<3><<<nb(n), 256, 0, st>>>(n, kp, c[s] * dt, b[s - 1], s == 1, b0, b1, m_s, kind_s, k4, S[s - 1], S[s], accx, accv);
        else
            k_rk_stage<2><<<nb(n), 256, 0, st>>>(n, kp, c[s] * dt, b[s - 1], s == 1, b0, b1, m_s, kind_s, k4, S[s - 1], S[s], accx, accv);
        }
    }
    // reverse sweep
    {
    KScope ks(ctx, SPH_K_RK, 1, st);
    if (kp.dim == 3) k_adj_gather<3><<<nb(n), 256, 0, st>>>(n, perm, x_bar, v_bar, rho_bar, yx, yv);
    else k_adj_gather<2><<<nb(n), 256, 0, st>>>(n, perm, x_bar, v_bar, rho_bar, yx, yv);
    }
    for (int s = 3; s >= 0; --s) {
        const float adt = s == 3 ? 0.f : c[s + 1] * dt;      // a_{s+1,s} = c_{s+1} in the classic tableau
        {
            KScope ks(ctx, SPH_K_RK, 1, st);
            k_adj_cot<<<nb(n), 256, 0, st>>>(n, b[s] * dt, adt, kind_s, yx, yv, Yx, Yv, cot, kbx);
        }
        SPH_TRY(sph_launch_vjp_sorted(ctx, kp, S[s].s0, S[s].s1, S[s].s2, cot, S[s].eos, nullptr, nullptr, nullptr, Yx, Yv,
                                      params_bar, 1, st));
        {
            KScope ks(ctx, SPH_K_RK, 1, st);
            k_adj_fix<<<nb(n), 256, 0, st>>>(n, s == 3, kbx, Yx, Yv, sumx, sumv);
        }
    }
    {
    KScope ks(ctx, SPH_K_RK, 1, st);
    if (kp.dim == 3) k_adj_final<3><<<nb(n), 256, 0, st>>>(n, perm, sumx, sumv, x_bar, v_bar, rho_bar);
    else k_adj_final<2><<<nb(n), 256, 0, st>>>(n, perm, sumx, sumv, x_bar, v_bar, rho_bar);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}
