// sph_delta.cu -- sph_params.delta_form = 1: the delta-SPH density diffusion of Antuono et al. [43],
// i.e. the Molteni-Colagrossi term of the RHS pair loop MINUS  delta l c0 sum_j V_j (g_i + g_j).(x_i - x_j) G  with
// g = <grad rho>^L the renormalised density gradient (Eq.44/45, reading R17), and its
// adjoint including the path through L_i.  Orchestration on top of a finished RHS / VJP launch, for the
// sorted state the pair kernels work on (so sph_rhs, sph_rhs_vjp and every RK stage of sph_rk_step(_vjp) get it):
//
//   forward   prep {x,y,z,h}, {V,rho}  ->  moments (pair pass)  ->  g = M^+ b per particle  ->  pair pass adding the term
//   adjoint   the same three, then the pair pass of the term's adjoint for lambda (x_bar, rho_bar, g_bar, sum lambda X),
//             g_bar through the per-particle adjoint of the pseudo-inverse and the renormalisation's adjoint pair pass
//             (x_bar, vol_bar, A_bar; vol = m/rho, A = rho), a combine pass, and delta_bar, c0_bar.
#include "sph_internal.cuh"

namespace {

inline unsigned nb256(int64_t n) { return (unsigned)((n + 255) / 256); }

// current positions with h, and {V, rho}, from the sorted state records (layouts: sph_pairs.cu load_part)
template <int DIM>
__global__ void k_delta_prep(int64_t n, const float4 *__restrict__ s0, const float4 *__restrict__ s1,
                             const float2 *__restrict__ s2, const float4 *__restrict__ cot, float4 *__restrict__ pos4,
                             float2 *__restrict__ va, float2 *__restrict__ lr)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float4 a = s0[p], b = s1[p];
    float V, rho, h;
    if (DIM == 3) {
        const float2 c = s2[p];
        pos4[p] = make_float4(a.x, a.y, a.z, c.y);
        V = c.x; rho = a.w; h = c.y;
    } else {
        pos4[p] = make_float4(a.x, a.y, 0.f, b.w);
        V = b.y; rho = b.x; h = b.w;
    }
    (void)h;
    va[p] = make_float2(V, rho);
    if (lr) lr[p] = make_float2(cot[p].x, rho);
}

// final outputs += direct part + path through the renormalised gradient:  x_bar += dx + x2,
// rho_bar += drho + A_bar - vol_bar V / rho   (vol = m/rho => d vol/d rho = -V/rho;  A = rho)
template <int DIM>
__global__ void k_delta_combine(int64_t n, const uint32_t *__restrict__ perm, const float4 *__restrict__ dx4,
                                const float *__restrict__ x2, const float *__restrict__ volb, const float *__restrict__ ab,
                                const float2 *__restrict__ va, float *__restrict__ xb, float *__restrict__ rb,
                                float4 *__restrict__ xb4)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float4 d = dx4[p];
    const float2 v = va[p];
    float add[3] = {d.x + x2[p * DIM], d.y + x2[p * DIM + 1], DIM == 3 ? d.z + x2[p * DIM + 2] : 0.f};
    const float addr = d.w + ab[p] - volb[p] * v.x / v.y;
    if (xb4) {
        float4 t = xb4[p];
        t.x += add[0]; t.y += add[1]; t.z += add[2]; t.w += addr;
        xb4[p] = t;
    } else {
        const int64_t i = perm[p];
#pragma unroll
        for (int k = 0; k < DIM; ++k) xb[i * DIM + k] += add[k];
        rb[i] += addr;
    }
}

// delta_bar += S / delta, c0_bar += S / c0 with S = sum_i lambda_i sum_j X_ij (fixed-order sum of the per-block partials)
__global__ void k_delta_params(int nblocks, const float *__restrict__ partial, float delta, float c0, float *__restrict__ params_bar)
{
    __shared__ double sh[128];
    double acc = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) acc += (double)partial[b];
    sh[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double S = 0.0;
        for (int t = 0; t < (int)blockDim.x; ++t) S += sh[t];
        if (delta != 0.f) params_bar[3] += (float)(S / (double)delta);
        params_bar[0] += (float)(S / (double)c0);
    }
}

int reserve_common(sph_ctx *ctx, int64_t n)
{
    SPH_TRY(ctx->d_pos.reserve((size_t)n * 16));
    SPH_TRY(ctx->d_va.reserve((size_t)n * 8));
    SPH_TRY(ctx->d_mom.reserve((size_t)n * 48));
    SPH_TRY(ctx->d_g4.reserve((size_t)n * 16));
    return SPH_OK;
}

// prep + moments + g; leaves {x,y,z,h} in d_pos, {V,rho} in d_va, the moments in d_mom, {g,V} in d_g4 (+ {lambda,rho} in d_lr)
int gradient_passes(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2, const float4 *cot,
                    cudaStream_t st)
{
    const int64_t n = ctx->n;
    SPH_TRY(reserve_common(ctx, n));
    if (cot) SPH_TRY(ctx->d_lr.reserve((size_t)n * 8));
    float4 *pos4 = ctx->d_pos.as<float4>();
    float2 *va = ctx->d_va.as<float2>(), *lr = cot ? ctx->d_lr.as<float2>() : nullptr;
    {
        KScope ks(ctx, SPH_K_PACK, 1, st);
        if (kp.dim == 3) k_delta_prep<3><<<nb256(n), 256, 0, st>>>(n, s0, s1, s2, cot, pos4, va, lr);
        else k_delta_prep<2><<<nb256(n), 256, 0, st>>>(n, s0, s1, s2, cot, pos4, va, lr);
    }
    KScope ks(ctx, SPH_K_DENSITY, 2, st);
    SPH_TRY(sph_renorm_moments_any(ctx, kp, pos4, va, ctx->d_mom.as<float4>(), st));
    SPH_TRY(sph_renorm_solve_sorted(ctx, kp, ctx->d_mom.as<float4>(), va, nullptr, ctx->d_g4.as<float4>(), nullptr, nullptr,
                                    nullptr, nullptr, st));
    return SPH_OK;
}

} // namespace

int sph_delta_forward(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2, float *drho,
                      float4 *out4, cudaStream_t st)
{
    SPH_TRY(gradient_passes(ctx, kp, s0, s1, s2, nullptr, st));
    KScope ks(ctx, SPH_K_RHS, 1, st);
    if (ctx->tile_mode)
        return sph_launch_delta_term_tile(ctx, kp, ctx->d_pos.as<float4>(), ctx->d_g4.as<float4>(), nullptr, false, drho, out4,
                                          nullptr, nullptr, nullptr, st);
    return sph_delta_term_generic(ctx, kp, ctx->d_pos.as<float4>(), ctx->d_g4.as<float4>(), nullptr, false, drho, out4, nullptr,
                                  nullptr, nullptr, nullptr, st);
}

int sph_delta_adjoint(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2, const float4 *cot,
                      float *xb, float *rb, float4 *xb4, float *params_bar, cudaStream_t st)
{
    const int64_t n = ctx->n;
    const int dim = kp.dim;
    SPH_TRY(gradient_passes(ctx, kp, s0, s1, s2, cot, st));
    SPH_TRY(ctx->d_dx4.reserve((size_t)n * 16));
    SPH_TRY(ctx->d_gb4.reserve((size_t)n * 16));
    SPH_TRY(ctx->d_rb.reserve((size_t)n * 16));
    SPH_TRY(ctx->d_rc.reserve((size_t)n * 16));
    SPH_TRY(ctx->d_rd.reserve((size_t)n * 8));
    SPH_TRY(ctx->d_re.reserve((size_t)n * 4));
    SPH_TRY(ctx->d_x2.reserve((size_t)n * 12));
    SPH_TRY(ctx->d_vb.reserve((size_t)n * 4));
    SPH_TRY(ctx->d_ab.reserve((size_t)n * 4));
    const float4 *pos4 = ctx->d_pos.as<float4>();
    int npart = ctx->tile_mode ? ctx->tg.ntiles : 0;
    if (!ctx->tile_mode) {
        // grid of the generic kernel (sph_delta_term_generic reports it); an upper bound sizes the buffer
        npart = (int)((n + 7) / 8) + 1;
    }
    SPH_TRY(ctx->d_part.reserve((size_t)npart * 4));
    {
        KScope ks(ctx, SPH_K_VJP, 1, st);
        if (ctx->tile_mode)
            SPH_TRY(sph_launch_delta_term_tile(ctx, kp, pos4, ctx->d_g4.as<float4>(), ctx->d_lr.as<float2>(), true, nullptr,
                                               nullptr, ctx->d_dx4.as<float4>(), ctx->d_gb4.as<float4>(),
                                               ctx->d_part.as<float>(), st));
        else
            SPH_TRY(sph_delta_term_generic(ctx, kp, pos4, ctx->d_g4.as<float4>(), ctx->d_lr.as<float2>(), true, nullptr,
                                           nullptr, ctx->d_dx4.as<float4>(), ctx->d_gb4.as<float4>(),
                                           ctx->d_part.as<float>(), &npart, st));
    }
    {
        KScope ks(ctx, SPH_K_VJP, 3, st);
        SPH_TRY(sph_renorm_solve_sorted(ctx, kp, ctx->d_mom.as<float4>(), ctx->d_va.as<float2>(), ctx->d_gb4.as<float4>(),
                                        nullptr, ctx->d_rb.as<float4>(), ctx->d_rc.as<float4>(), ctx->d_rd.as<float2>(),
                                        ctx->d_re.as<float>(), st));
        SPH_TRY(sph_renorm_vjp_pairs_any(ctx, kp, pos4, ctx->d_rb.as<float4>(), ctx->d_rc.as<float4>(), ctx->d_rd.as<float2>(),
                                         ctx->d_re.as<float>(), nullptr, ctx->d_x2.as<float>(), ctx->d_vb.as<float>(),
                                         ctx->d_ab.as<float>(), st));
        if (dim == 3)
            k_delta_combine<3><<<nb256(n), 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), ctx->d_dx4.as<float4>(),
                                                         ctx->d_x2.as<float>(), ctx->d_vb.as<float>(), ctx->d_ab.as<float>(),
                                                         ctx->d_va.as<float2>(), xb, rb, xb4);
        else
            k_delta_combine<2><<<nb256(n), 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), ctx->d_dx4.as<float4>(),
                                                         ctx->d_x2.as<float>(), ctx->d_vb.as<float>(), ctx->d_ab.as<float>(),
                                                         ctx->d_va.as<float2>(), xb, rb, xb4);
    }
    if (params_bar) {
        KScope ks(ctx, SPH_K_REDUCE, 1, st);
        k_delta_params<<<1, 128, 0, st>>>(npart, ctx->d_part.as<float>(), kp.delta, kp.c0, params_bar);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}
