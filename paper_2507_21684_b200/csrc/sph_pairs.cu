// sph_pairs.cu -- the pair-sum kernels: D (density), R0 (EOS prologue / pack), R1 (RHS), B1 (VJP), B2 (parameter
// reduction) of SURVEY.md 8(a).  Gather formulation: a group of GS lanes owns a row, strides over the row's CSR
// entries (coalesced index reads), gathers the neighbour's sorted float4 state, and reduces with shuffles.
// No float atomics anywhere; every sum has a fixed order for a given launch configuration.
//
// Formulas: include/sph.h header comment and DESIGN.md section 2 (Eq.8, 9, 12, 40, 42, 7).
#include "sph_internal.cuh"
#include "sph_pair_math.cuh"

#include <math.h>

namespace {

constexpr int kBlock = 256;          // threads per block
constexpr int kRowsPerGroup = 8;     // rows each lane group walks through

// global-memory load of a particle record (layout: sph_pair_math.cuh)
template <int DIM>
__device__ __forceinline__ Part load_part(const float4 *__restrict__ s0, const float4 *__restrict__ s1,
                                          const float2 *__restrict__ s2, int64_t j)
{
    const float4 a = __ldg(s0 + j), b = __ldg(s1 + j);
    if (DIM == 3) {
        const float2 c = __ldg(s2 + j);
        return part_unpack<3>(a, b, c.x, c.y);
    }
    return part_unpack<DIM>(a, b);
}

template <int DIM, bool WRAP>
__device__ __forceinline__ void rel_pos(const float *xi, const float *xj, const KPar &kp, float *d, float &r2)
{
    r2 = 0.f;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        float dk = xi[k] - xj[k];
        if (WRAP && kp.periodic[k]) dk = dk > kp.halfL[k] ? dk - kp.L[k] : (dk < -kp.halfL[k] ? dk + kp.L[k] : dk);
        d[k] = dk;
        r2 = fmaf(dk, dk, r2);
    }
    if (DIM == 2) d[2] = 0.f;
}

// does this row need the minimum-image test?  (only rows within `margin` of a periodic face can see the seam)
__device__ __forceinline__ bool row_near_seam(const float *xi, const KPar &kp, float margin)
{
    bool s = false;
    for (int k = 0; k < kp.dim; ++k)
        if (kp.periodic[k]) s = s || (xi[k] - kp.lo[k] < margin) || (kp.hi[k] - xi[k] < margin);
    return s;
}

// Sum over the GS lanes that share a row.  The shuffles name only the lanes of the group: groups of one warp leave
// the row loop at different times (row >= n in the last block), so a full-warp mask would be undefined there.
template <int GS>
__device__ __forceinline__ float group_sum(float v)
{
    const uint32_t gmask = (0xffffffffu >> (32 - GS)) << ((threadIdx.x & 31u) & ~(uint32_t)(GS - 1));
#pragma unroll
    for (int o = GS / 2; o > 0; o >>= 1) v += __shfl_xor_sync(gmask, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------ R0: pack + EOS
// Gathers the caller's arrays into the sorted SoA, wraps positions (R4), evaluates the Tait EOS (PAPER.md:112
// Eq.12) as p = B expm1(gamma log1p((rho-rho0)/rho0)) so that small compressions keep full relative accuracy.
template <int DIM>
__global__ void k_pack_state(int64_t n, KPar kp, const uint32_t *__restrict__ perm, const float4 *__restrict__ pos_s,
                             const float *__restrict__ x, const float *__restrict__ v, const float *__restrict__ rho,
                             const float *__restrict__ m, const uint8_t *__restrict__ kind,
                             float4 *__restrict__ s0, float4 *__restrict__ s1, float2 *__restrict__ s2,
                             float4 *__restrict__ eos, uint8_t *__restrict__ kind_s, uint32_t *__restrict__ um)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    // um[0] (preset to non-zero): cleared when the masses are not all equal; um[1] = the common mass (bits of m[0])
    const float m_first = __ldg(m);
    if (p == 0) um[1] = __float_as_uint(m_first);
    const float4 pb = pos_s[p];                           // wrapped build position, h
    const float xb[3] = {pb.x, pb.y, pb.z};
    float xw[3] = {0.f, 0.f, 0.f}, vv[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        float xv = x[i * DIM + k];
        if (kp.periodic[k]) {
            // the periodic image next to the build position: a particle that drifted across a face since the
            // build stays in the frame of its build cell (the tile kernels shift whole halo cells, not pairs)
            xv = wrap_coord(xv, kp.lo[k], kp.hi[k], kp.L[k]);
            const float dd = xv - xb[k];
            xv = dd > kp.halfL[k] ? xv - kp.L[k] : (dd < -kp.halfL[k] ? xv + kp.L[k] : xv);
        }
        xw[k] = xv;
        vv[k] = v[i * DIM + k];
    }
    const float r = rho[i], mi = m[i], h = pb.w;
    if (mi != m_first) um[0] = 0u;
    sph_flag_bad_state(um, r, mi);
    const float u = (r - kp.rho0) / kp.rho0;
    const float lg = log1pf(u);
    const float ugm1 = expm1f(kp.gamma * lg);        // (rho/rho0)^gamma - 1
    const float ug = ugm1 + 1.0f;
    const float pr = kp.Bp * ugm1;                    // Tait pressure
    const float ir = 1.0f / r, ir2 = ir * ir;
    const float V = mi * ir, P = pr * ir2;
    if (DIM == 3) {
        s0[p] = make_float4(xw[0], xw[1], xw[2], r);
        s1[p] = make_float4(vv[0], vv[1], vv[2], P);
        s2[p] = make_float2(V, h);
    } else {
        s0[p] = make_float4(xw[0], xw[1], vv[0], vv[1]);
        s1[p] = make_float4(r, V, P, h);
    }
    if (eos) {
        // derivatives of P = p/rho^2 needed by the adjoint of the EOS prologue
        const float dp_drho = kp.c0 * kp.c0 * ug / (1.0f + u);                     // c0^2 (rho/rho0)^(gamma-1)
        const float dP = dp_drho * ir2 - 2.0f * pr * ir2 * ir;
        const float dp_drho0 = kp.c0 * kp.c0 / kp.gamma * ugm1 - kp.c0 * kp.c0 * ug;
        const float dp_dgam = -kp.Bp / kp.gamma * ugm1 + kp.Bp * ug * lg;
        eos[p] = make_float4(dP, dp_drho0 * ir2, dp_dgam * ir2, mi);
    }
    kind_s[p] = kind[i];
}

__global__ void k_pack_cot(int64_t n, int dim, const uint32_t *__restrict__ perm, const uint8_t *__restrict__ kind_s,
                           const float *__restrict__ lam, const float *__restrict__ mu, float4 *__restrict__ cot)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    float m0 = mu[i * dim], m1 = mu[i * dim + 1], m2 = dim == 3 ? mu[i * dim + 2] : 0.f;
    if (kind_s[p]) m0 = m1 = m2 = 0.f;                 // a_i = 0 for boundary kinds => mu_i has no effect
    cot[p] = make_float4(lam[i], m0, m1, m2);
}

__global__ void k_gather_f32(int64_t n, const uint32_t *__restrict__ perm, const float *__restrict__ in,
                             float *__restrict__ out)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) out[p] = in[perm[p]];
}
// the same, and clears *um (preset to non-zero) when the values are not all equal to in[0]
__global__ void k_gather_f32_um(int64_t n, const uint32_t *__restrict__ perm, const float *__restrict__ in,
                                float *__restrict__ out, uint32_t *__restrict__ um)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float first = __ldg(in), v = in[perm[p]];
    out[p] = v;
    if (v != first) *um = 0u;
}
__global__ void k_gather_f32_w(int64_t n, const uint32_t *__restrict__ perm, const float *__restrict__ in,
                               float4 *__restrict__ out)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) out[p] = make_float4(0.f, 0.f, 0.f, in[perm[p]]);
}

// ------------------------------------------------------------------------------------------ D: density
template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kBlock)
k_density(int64_t n, KPar kp, float margin, const float4 *__restrict__ pos_s, const float *__restrict__ m_s,
          const long long *__restrict__ row_ptr, const int32_t *__restrict__ col, const uint32_t *__restrict__ perm,
          float *__restrict__ rho_out)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const float4 pi = __ldg(pos_s + row);
        const float xi[3] = {pi.x, pi.y, pi.z};
        const bool seam = row_near_seam(xi, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        float acc = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const float4 pj = __ldg(pos_s + j);
            const float xj[3] = {pj.x, pj.y, pj.z};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(xi, xj, kp, d, r2); else rel_pos<DIM, false>(xi, xj, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);
            const float t2 = t * t, t6 = t2 * t2 * t2;
            const float w = hc.cW * t6 * fmaf(q, fmaf(q, 35.0f / 3.0f, 6.0f), 1.0f);   // Eq.25/27
            acc = fmaf(__ldg(m_s + j), w, acc);
        }
        acc = group_sum<GS>(acc);
        if (gl == 0) rho_out[perm[row]] = acc;
    }
}

// ------------------------------------------------------------------------------------------ D^T: density adjoint
// x_bar_i = sum_j (rb_i m_j + rb_j m_i) G_ij d_ij,  m_bar_i = sum_j rb_j W_ij   (include/sph.h sph_density_vjp)
__global__ void k_gather_f32x2(int64_t n, const uint32_t *__restrict__ perm, const float *__restrict__ a,
                               const float *__restrict__ b, float2 *__restrict__ out)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) {
        const int64_t i = perm[p];
        out[p] = make_float2(a[i], b[i]);
    }
}

template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kBlock)
k_density_vjp(int64_t n, KPar kp, float margin, const float4 *__restrict__ pos_s, const float2 *__restrict__ mr_s,
              const long long *__restrict__ row_ptr, const int32_t *__restrict__ col, const uint32_t *__restrict__ perm,
              float *__restrict__ xb_out, float *__restrict__ mb_out)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const float4 pi = __ldg(pos_s + row);
        const float2 ai = __ldg(mr_s + row);                  // {m_i, rho_bar_i}
        const float xi[3] = {pi.x, pi.y, pi.z};
        const bool seam = row_near_seam(xi, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        float x0 = 0.f, x1 = 0.f, x2 = 0.f, mb = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const float4 pj = __ldg(pos_s + j);
            const float2 aj = __ldg(mr_s + j);
            const float xj[3] = {pj.x, pj.y, pj.z};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(xi, xj, kp, d, r2); else rel_pos<DIM, false>(xi, xj, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                               // Eq.29
            const float w = hc.cW * (t4 * t2) * fmaf(q, fmaf(q, 35.0f / 3.0f, 6.0f), 1.0f);       // Eq.25/27
            const float c = fmaf(ai.y, aj.x, aj.y * ai.x) * G;
            x0 = fmaf(c, d[0], x0);
            x1 = fmaf(c, d[1], x1);
            if (DIM == 3) x2 = fmaf(c, d[2], x2);
            mb = fmaf(aj.y, w, mb);
        }
        x0 = group_sum<GS>(x0);
        x1 = group_sum<GS>(x1);
        if (DIM == 3) x2 = group_sum<GS>(x2);
        mb = group_sum<GS>(mb);
        if (gl == 0) {
            const int64_t i = perm[row];
            xb_out[i * DIM] = x0;
            xb_out[i * DIM + 1] = x1;
            if (DIM == 3) xb_out[i * DIM + 2] = x2;
            if (mb_out) mb_out[i] = mb;
        }
    }
}

// ------------------------------------------------------------------------------------------ kernel-gradient sum
// g_i = sum_j a_j G_ij d_ij and its adjoint (include/sph.h sph_grad_sum / sph_grad_sum_vjp; Eq.24)
template <int DIM>
__global__ void k_gather_vec_a(int64_t n, const uint32_t *__restrict__ perm, const float *__restrict__ vec,
                               const float *__restrict__ a, float4 *__restrict__ out)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) {
        const int64_t i = perm[p];
        out[p] = make_float4(vec[i * DIM], vec[i * DIM + 1], DIM == 3 ? vec[i * DIM + 2] : 0.f, a[i]);
    }
}

// VJP = false: GA.w = a (xyz unused), writes g;  VJP = true: GA = {g_bar, a}, writes x_bar and a_bar
template <int DIM, int GS, bool VARH, bool VJP>
__global__ void __launch_bounds__(kBlock)
k_grad_sum(int64_t n, KPar kp, float margin, const float4 *__restrict__ pos_s, const float4 *__restrict__ ga_s,
           const long long *__restrict__ row_ptr, const int32_t *__restrict__ col, const uint32_t *__restrict__ perm,
           float *__restrict__ v_out, float *__restrict__ a_out)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const float4 pi = __ldg(pos_s + row);
        const float4 gi = __ldg(ga_s + row);
        const float xi[3] = {pi.x, pi.y, pi.z};
        const bool seam = row_near_seam(xi, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        float x0 = 0.f, x1 = 0.f, x2 = 0.f, ab = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const float4 pj = __ldg(pos_s + j);
            const float4 gj = __ldg(ga_s + j);
            const float xj[3] = {pj.x, pj.y, pj.z};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(xi, xj, kp, d, r2); else rel_pos<DIM, false>(xi, xj, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                               // Eq.29
            if (!VJP) {
                const float c = gj.w * G;
                x0 = fmaf(c, d[0], x0);
                x1 = fmaf(c, d[1], x1);
                if (DIM == 3) x2 = fmaf(c, d[2], x2);
            } else {
                const float K = hc.cK * t4;                                                       // Eq.16
                const float dgi = fmaf(d[2], gi.z, fmaf(d[1], gi.y, d[0] * gi.x));
                const float dgj = fmaf(d[2], gj.z, fmaf(d[1], gj.y, d[0] * gj.x));
                const float cG = G * gj.w, cGp = G * gi.w;                    // a_j G, a_i G
                const float cd = K * fmaf(gj.w, dgi, -(gi.w * dgj));          // K (a_j d.gb_i - a_i d.gb_j)
                x0 += fmaf(cG, gi.x, fmaf(-cGp, gj.x, cd * d[0]));
                x1 += fmaf(cG, gi.y, fmaf(-cGp, gj.y, cd * d[1]));
                if (DIM == 3) x2 += fmaf(cG, gi.z, fmaf(-cGp, gj.z, cd * d[2]));
                ab = fmaf(-G, dgj, ab);
            }
        }
        x0 = group_sum<GS>(x0);
        x1 = group_sum<GS>(x1);
        if (DIM == 3) x2 = group_sum<GS>(x2);
        if (VJP) ab = group_sum<GS>(ab);
        if (gl == 0) {
            const int64_t i = perm[row];
            v_out[i * DIM] = x0;
            v_out[i * DIM + 1] = x1;
            if (DIM == 3) v_out[i * DIM + 2] = x2;
            if (VJP && a_out) a_out[i] = ab;
        }
    }
}

// ------------------------------------------------------------------------------------------ kernel renormalisation
// PAPER.md:524-528 Eq.44/45 (include/sph.h sph_renorm_gradient).  The pair pass accumulates the symmetric matrix
// M_i = sum_j V_j (x_j - x_i) (x) grad_i W_ij = -sum_j V_j G_ij d d^T and b_i = sum_j V_j (A_j - A_i) G_ij d into a
// sorted-order record of kRenormRec<DIM> float4 per row; k_renorm_solve then takes L_i = M_i^+ and L_i b_i with one
// thread per particle (the eigen-solve would otherwise serialise on one lane of every row group).
// record: 3D {xx,xy,xz,yy} {yz,zz,b0,b1} {b2,-,-,-};  2D {xx,xy,yy,b0} {b1,-,-,-}
template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kBlock)
k_renorm(int64_t n, KPar kp, float margin, const float4 *__restrict__ pos_s, const float2 *__restrict__ va_s,
         const long long *__restrict__ row_ptr, const int32_t *__restrict__ col, float4 *__restrict__ mom)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const float4 pi = __ldg(pos_s + row);
        const float Ai = __ldg(va_s + row).y;
        const float xi[3] = {pi.x, pi.y, pi.z};
        const bool seam = row_near_seam(xi, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        float mxx = 0.f, mxy = 0.f, mxz = 0.f, myy = 0.f, myz = 0.f, mzz = 0.f, b0 = 0.f, b1 = 0.f, b2 = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const float4 pj = __ldg(pos_s + j);
            const float2 aj = __ldg(va_s + j);                  // {V_j, A_j}
            const float xj[3] = {pj.x, pj.y, pj.z};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(xi, xj, kp, d, r2); else rel_pos<DIM, false>(xi, xj, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                               // Eq.29
            const float c = aj.x * G, dA = aj.y - Ai;
            const float c0 = c * d[0], c1 = c * d[1], c2 = c * d[2];
            mxx = fmaf(-c0, d[0], mxx);
            mxy = fmaf(-c0, d[1], mxy);
            myy = fmaf(-c1, d[1], myy);
            b0 = fmaf(c0, dA, b0);
            b1 = fmaf(c1, dA, b1);
            if (DIM == 3) {
                mxz = fmaf(-c0, d[2], mxz);
                myz = fmaf(-c1, d[2], myz);
                mzz = fmaf(-c2, d[2], mzz);
                b2 = fmaf(c2, dA, b2);
            }
        }
        mxx = group_sum<GS>(mxx); mxy = group_sum<GS>(mxy); myy = group_sum<GS>(myy);
        b0 = group_sum<GS>(b0); b1 = group_sum<GS>(b1);
        if (DIM == 3) {
            mxz = group_sum<GS>(mxz); myz = group_sum<GS>(myz); mzz = group_sum<GS>(mzz); b2 = group_sum<GS>(b2);
        }
        if (gl == 0) {
            if (DIM == 3) {
                mom[row * 3] = make_float4(mxx, mxy, mxz, myy);
                mom[row * 3 + 1] = make_float4(myz, mzz, b0, b1);
                mom[row * 3 + 2] = make_float4(b2, 0.f, 0.f, 0.f);
            } else {
                mom[row * 2] = make_float4(mxx, mxy, myy, b0);
                mom[row * 2 + 1] = make_float4(b1, 0.f, 0.f, 0.f);
            }
        }
    }
}

// Moore-Penrose inverse of a symmetric matrix by its eigen-decomposition: eigenvalues with |lambda| <= rcond * max|lambda|
// are dropped ("pseudo-inverse for numerical stability"; explicit in 2D as in the paper, cyclic Jacobi in 3D)
__device__ __forceinline__ void jacobi_rotate(float &app, float &aqq, float &apq, float &arp, float &arq,
                                              float (&V)[3][3], int p, int q)
{
    if (fabsf(apq) <= 1e-30f) return;
    const float theta = (aqq - app) / (2.0f * apq);
    const float t = copysignf(1.0f, theta) / (fabsf(theta) + sqrtf(fmaf(theta, theta, 1.0f)));
    const float c = rsqrtf(fmaf(t, t, 1.0f)), s = t * c;
    app = fmaf(-t, apq, app);
    aqq = fmaf(t, apq, aqq);
    apq = 0.f;
    const float rp = arp, rq = arq;                             // the third row/column r
    arp = c * rp - s * rq;
    arq = s * rp + c * rq;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float vp = V[k][p], vq = V[k][q];
        V[k][p] = c * vp - s * vq;
        V[k][q] = s * vp + c * vq;
    }
}

// L = M^+ and P = projector on the range of M (sum of v v^T over the retained eigenvectors), M symmetric given as
// {xx, xy, xz, yy, yz, zz} (2D: xz = yz = zz = 0 and only the upper-left 2x2 of L, P is meaningful)
template <int DIM>
__device__ __forceinline__ void renorm_pinv(const float (&m)[6], float rcond, float (&L)[3][3], float (&P)[3][3])
{
    float lam[3] = {0.f, 0.f, 0.f};
    float V[3][3] = {{1.f, 0.f, 0.f}, {0.f, 1.f, 0.f}, {0.f, 0.f, 1.f}};
    if (DIM == 2) {
        const float a = m[0], b = m[1], c = m[3];
        const float hd = 0.5f * (a - c), rad = sqrtf(fmaf(hd, hd, b * b)), mid = 0.5f * (a + c);
        lam[0] = mid + rad;
        lam[1] = mid - rad;
        // unit eigenvector of lam[0]: (cos, sin) of half the angle of (a - c, 2b)
        float cs = 1.f, sn = 0.f;
        if (rad > 0.f) {
            const float cx = hd / rad, sx = b / rad;            // cos, sin of the full angle
            // the larger of the two from the half-angle formula (no cancellation), the other from sin(2p) = 2 sin cos
            if (cx >= 0.f) {
                cs = sqrtf(0.5f * (1.0f + cx));
                sn = sx / (2.0f * cs);
            } else {
                sn = copysignf(sqrtf(0.5f * (1.0f - cx)), b);
                cs = sx / (2.0f * sn);
            }
        }
        V[0][0] = cs; V[1][0] = sn; V[0][1] = -sn; V[1][1] = cs;
    } else {
        float axx = m[0], axy = m[1], axz = m[2], ayy = m[3], ayz = m[4], azz = m[5];
#pragma unroll 1
        for (int sweep = 0; sweep < 6; ++sweep) {
            jacobi_rotate(axx, ayy, axy, axz, ayz, V, 0, 1);
            jacobi_rotate(axx, azz, axz, axy, ayz, V, 0, 2);
            jacobi_rotate(ayy, azz, ayz, axy, axz, V, 1, 2);
        }
        lam[0] = axx; lam[1] = ayy; lam[2] = azz;
    }
    const float cut = rcond * fmaxf(fabsf(lam[0]), fmaxf(fabsf(lam[1]), fabsf(lam[2])));
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) L[r][c] = P[r][c] = 0.f;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        const bool keep = fabsf(lam[k]) > cut;
        const float inv = keep ? 1.0f / lam[k] : 0.f, one = keep ? 1.0f : 0.f;
#pragma unroll
        for (int r = 0; r < DIM; ++r)
#pragma unroll
            for (int c = 0; c < DIM; ++c) {
                L[r][c] = fmaf(inv * V[r][k], V[c][k], L[r][c]);
                P[r][c] = fmaf(one * V[r][k], V[c][k], P[r][c]);
            }
    }
}

template <int DIM>
__device__ __forceinline__ void renorm_load(const float4 *__restrict__ mom, int64_t p, float (&m)[6], float (&b)[3])
{
    if (DIM == 2) {
        const float4 r0 = mom[p * 2];
        m[0] = r0.x; m[1] = r0.y; m[2] = 0.f; m[3] = r0.z; m[4] = 0.f; m[5] = 0.f;
        b[0] = r0.w; b[1] = mom[p * 2 + 1].x; b[2] = 0.f;
    } else {
        const float4 r0 = mom[p * 3], r1 = mom[p * 3 + 1];
        m[0] = r0.x; m[1] = r0.y; m[2] = r0.z; m[3] = r0.w; m[4] = r1.x; m[5] = r1.y;
        b[0] = r1.z; b[1] = r1.w; b[2] = mom[p * 3 + 2].x;
    }
}

template <int DIM>
__global__ void k_renorm_solve(int64_t n, const float4 *__restrict__ mom, const uint32_t *__restrict__ perm, float rcond,
                               float *__restrict__ L_out, float *__restrict__ grad_out)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    float m[6], b[3], L[3][3], P[3][3];
    renorm_load<DIM>(mom, p, m, b);
    renorm_pinv<DIM>(m, rcond, L, P);
    if (L_out)
#pragma unroll
        for (int r = 0; r < DIM; ++r)
#pragma unroll
            for (int c = 0; c < DIM; ++c) L_out[i * DIM * DIM + r * DIM + c] = L[r][c];
    if (grad_out)
#pragma unroll
        for (int r = 0; r < DIM; ++r) grad_out[i * DIM + r] = fmaf(L[r][0], b[0], fmaf(L[r][1], b[1], L[r][2] * b[2]));
}

// Adjoint of g = M^+ b per particle (include/sph.h sph_renorm_gradient_vjp): b_bar = L g_bar and, with the differential of
// the pseudo-inverse at constant rank, M_bar = -b_bar g^T + ((I - P) g_bar) (L g)^T.  Only N = M_bar + M_bar^T enters the
// pair terms.  Writes the sorted records the pair pass gathers:
//   rb = {V, A, b_bar0, b_bar1};  3D: rc = {b_bar2, Nxx, Nxy, Nxz}, rd = {Nyy, Nyz}, re = Nzz;  2D: rd = {Nxx, Nxy}, re = Nyy
template <int DIM>
__global__ void k_renorm_solve_vjp(int64_t n, const float4 *__restrict__ mom, const float2 *__restrict__ va_s,
                                   const uint32_t *__restrict__ perm, const float *__restrict__ grad_bar, float rcond,
                                   float4 *__restrict__ rb, float4 *__restrict__ rc, float2 *__restrict__ rd,
                                   float *__restrict__ re)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    float m[6], b[3], L[3][3], P[3][3];
    renorm_load<DIM>(mom, p, m, b);
    renorm_pinv<DIM>(m, rcond, L, P);
    float gb[3] = {grad_bar[i * DIM], grad_bar[i * DIM + 1], DIM == 3 ? grad_bar[i * DIM + 2] : 0.f};
    float g[3], bb[3], c[3], u[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        g[r] = fmaf(L[r][0], b[0], fmaf(L[r][1], b[1], L[r][2] * b[2]));
        bb[r] = fmaf(L[r][0], gb[0], fmaf(L[r][1], gb[1], L[r][2] * gb[2]));
        c[r] = gb[r] - fmaf(P[r][0], gb[0], fmaf(P[r][1], gb[1], P[r][2] * gb[2]));
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) u[r] = fmaf(L[r][0], g[0], fmaf(L[r][1], g[1], L[r][2] * g[2]));
    auto N = [&](int r, int s) { return -(bb[r] * g[s] + g[r] * bb[s]) + (c[r] * u[s] + u[r] * c[s]); };
    const float2 va = va_s[p];
    rb[p] = make_float4(va.x, va.y, bb[0], bb[1]);
    if (DIM == 3) {
        rc[p] = make_float4(bb[2], N(0, 0), N(0, 1), N(0, 2));
        rd[p] = make_float2(N(1, 1), N(1, 2));
        re[p] = N(2, 2);
    } else {
        rd[p] = make_float2(N(0, 0), N(0, 1));
        re[p] = N(1, 1);
    }
}

// Pair pass of the adjoint, gather form over the symmetric list: row i evaluates the ordered pairs (i <- j) and (j <- i)
// and keeps what lands on i.  With d = x_i - x_j, dA = A_j - A_i, a_i = d^T M_bar_i d = (d^T N_i d)/2, be_i = b_bar_i . d:
//   F_ij = V_j [ -K a_i d - G N_i d + dA (K be_i d + G b_bar_i) ],   F_ji = V_i [ K a_j d + G N_j d - dA (K be_j d + G b_bar_j) ]
//   x_bar_i = sum_j F_ij - F_ji,   vol_bar_i = sum_j G (-a_j + dA be_j),   A_bar_i = -sum_j G (V_i be_j + V_j be_i)
template <int DIM, int GS, bool VARH>
__global__ void __launch_bounds__(kBlock)
k_renorm_vjp(int64_t n, KPar kp, float margin, const float4 *__restrict__ pos_s, const float4 *__restrict__ rb,
             const float4 *__restrict__ rc, const float2 *__restrict__ rd, const float *__restrict__ re,
             const long long *__restrict__ row_ptr, const int32_t *__restrict__ col, const uint32_t *__restrict__ perm,
             float *__restrict__ xb_out, float *__restrict__ vb_out, float *__restrict__ ab_out)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const float4 pi = __ldg(pos_s + row);
        const RenormRec ri = renorm_rec<DIM>(__ldg(rb + row), DIM == 3 ? __ldg(rc + row) : make_float4(0.f, 0.f, 0.f, 0.f),
                                             __ldg(rd + row), __ldg(re + row));
        const float xi[3] = {pi.x, pi.y, pi.z};
        const bool seam = row_near_seam(xi, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        float xb[3] = {0.f, 0.f, 0.f}, vb = 0.f, ab = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const float4 pj = __ldg(pos_s + j);
            const RenormRec rj = renorm_rec<DIM>(__ldg(rb + j), DIM == 3 ? __ldg(rc + j) : make_float4(0.f, 0.f, 0.f, 0.f),
                                                 __ldg(rd + j), __ldg(re + j));
            const float xj[3] = {pj.x, pj.y, pj.z};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(xi, xj, kp, d, r2); else rel_pos<DIM, false>(xi, xj, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);                               // Eq.29
            const float K = hc.cK * t4;                                                           // Eq.16
            renorm_vjp_pair<DIM>(ri, rj, d, G, K, xb, vb, ab);
        }
#pragma unroll
        for (int k = 0; k < DIM; ++k) xb[k] = group_sum<GS>(xb[k]);
        vb = group_sum<GS>(vb);
        ab = group_sum<GS>(ab);
        if (gl == 0) {
            const int64_t i = perm ? (int64_t)perm[row] : row;       // null perm: sorted order
#pragma unroll
            for (int k = 0; k < DIM; ++k) xb_out[i * DIM + k] = xb[k];
            if (vb_out) vb_out[i] = vb;
            if (ab_out) ab_out[i] = ab;
        }
    }
}

// ------------------------------------------------------------------------------------------ R1: RHS
// OUT_SORTED: write float4 {a, drho/dt} in sorted order (RK stages); else scatter to the caller's arrays.
template <int DIM, int GS, bool VARH, bool OUT_SORTED>
__global__ void __launch_bounds__(kBlock)
k_rhs(int64_t n, KPar kp, float margin, const float4 *__restrict__ s0, const float4 *__restrict__ s1,
      const float2 *__restrict__ s2, const uint8_t *__restrict__ kind_s, const long long *__restrict__ row_ptr,
      const int32_t *__restrict__ col, const uint32_t *__restrict__ perm, float *__restrict__ drho_out,
      float *__restrict__ acc_out, float4 *__restrict__ out4)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const Part pi = load_part<DIM>(s0, s1, s2, row);
        const bool seam = row_near_seam(pi.x, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        const float visc_i = kp.rho0 / pi.rho;            // rho0/rho_i of the viscous term
        float sA = 0.f, sD = 0.f, a0 = 0.f, a1 = 0.f, a2 = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const Part pj = load_part<DIM>(s0, s1, s2, j);
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(pi.x, pj.x, kp, d, r2); else rel_pos<DIM, false>(pi.x, pj.x, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.h, pj.h), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);          // kernel clamp: skin pairs contribute exactly 0
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);
            float s = (pi.v[0] - pj.v[0]) * d[0];
            s = fmaf(pi.v[1] - pj.v[1], d[1], s);
            if (DIM == 3) s = fmaf(pi.v[2] - pj.v[2], d[2], s);
            const float invR = fast_rcp(r2 + hc.e2);
            const float VG = pj.V * G;
            // continuity (Eq.9, physical sign) and delta-term (Brookshaw Laplacian of rho)
            sA = fmaf(VG, s, sA);
            const float dterm = VG * (pi.rho - pj.rho) * (r2 * invR);
            sD = VARH ? fmaf(hc.kd, dterm, sD) : sD + dterm;
            // pressure (Eq.40, symmetric) + viscosity (Eq.7 with the delta-SPH Pi_ij)
            // pressure pair factor e: P_i + P_j (form 0, Eq.40) or (p_i + p_j)/(rho_i rho_j) (form 1)
            const float epair = kp.form == 0 ? pi.P + pj.P
                                             : fmaf(pi.P * pi.rho, fast_rcp(pj.rho), pj.P * pj.rho * (visc_i / kp.rho0));
            const float E = -(pj.V * pj.rho) * epair;
            const float Phi = hc.eta * visc_i * pj.V * s * invR;
            const float cf = (E + Phi) * G;
            a0 = fmaf(cf, d[0], a0);
            a1 = fmaf(cf, d[1], a1);
            if (DIM == 3) a2 = fmaf(cf, d[2], a2);
        }
        float dr = pi.rho * sA + (VARH ? sD : hu.kd * sD);
        dr = group_sum<GS>(dr);
        a0 = group_sum<GS>(a0);
        a1 = group_sum<GS>(a1);
        if (DIM == 3) a2 = group_sum<GS>(a2);
        if (gl == 0) {
            const bool fixed = kind_s[row] != 0;
            a0 = fixed ? 0.f : a0 + kp.g[0];
            a1 = fixed ? 0.f : a1 + kp.g[1];
            a2 = fixed ? 0.f : a2 + kp.g[2];
            if (OUT_SORTED) {
                out4[row] = make_float4(a0, a1, a2, dr);
            } else {
                const int64_t i = perm[row];
                drho_out[i] = dr;
                acc_out[i * DIM] = a0;
                acc_out[i * DIM + 1] = a1;
                if (DIM == 3) acc_out[i * DIM + 2] = a2;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ B1: VJP
// Row i evaluates BOTH ordered pairs (i<-j) and (j<-i) of every neighbour j and keeps what lands on i
// (possible because the list is symmetric), so there is no scatter.  The pressure enters through the
// per-particle P_i = p_i/rho_i^2: its adjoint is collected as Z_i and pushed through the EOS once per row.
// Per-lane running sums of the scalar-parameter partials are reduced per block in a fixed order (B2).
constexpr int kNPart = 12;   // S_D1, S_Phi1, S_PhiL, S_eps, T_E, T_rho0, T_gam, g0, g1, g2, (2 spare)

template <int DIM, int GS, bool VARH, bool OUT_SORTED>
__global__ void __launch_bounds__(kBlock)
k_vjp(int64_t n, KPar kp, float margin, const float4 *__restrict__ s0, const float4 *__restrict__ s1,
      const float2 *__restrict__ s2, const float4 *__restrict__ cot, const float4 *__restrict__ eos,
      const long long *__restrict__ row_ptr, const int32_t *__restrict__ col, const uint32_t *__restrict__ perm,
      float *__restrict__ xb_out, float *__restrict__ vb_out, float *__restrict__ rb_out,
      float4 *__restrict__ xb4, float4 *__restrict__ vb4, float *__restrict__ partials)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    float S_D1 = 0.f, S_P1 = 0.f, S_PL = 0.f, S_eps = 0.f;       // per lane, over all its pairs
    float T_E = 0.f, T_0 = 0.f, T_g = 0.f, G0 = 0.f, G1 = 0.f, G2 = 0.f;   // lane 0 of each group, per row
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const Part pi = load_part<DIM>(s0, s1, s2, row);
        const float4 ci = __ldg(cot + row);
        const float4 ei = __ldg(eos + row);                    // {dP/drho, dP/drho0, dP/dgamma, m}
        const float lam_i = ci.x, mu_i[3] = {ci.y, ci.z, ci.w};
        const float m_i = ei.w;
        const bool seam = row_near_seam(pi.x, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        const float ir_i = 1.0f / pi.rho;
        float xb[3] = {0.f, 0.f, 0.f}, vb[3] = {0.f, 0.f, 0.f}, rb = 0.f, Z = 0.f, Zr = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const Part pj = load_part<DIM>(s0, s1, s2, j);
            const float4 cj = __ldg(cot + j);
            const float lam_j = cj.x, mu_j[3] = {cj.y, cj.z, cj.w};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(pi.x, pj.x, kp, d, r2); else rel_pos<DIM, false>(pi.x, pj.x, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.h, pj.h), kp);
            const float q = fast_sqrt(r2) * hc.invH;
            const float t = fmaxf(1.0f - q, 0.f);
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f, q, 1.0f) * (t4 * t);
            const float K = hc.cK * t4;
            float w[3] = {pi.v[0] - pj.v[0], pi.v[1] - pj.v[1], DIM == 3 ? pi.v[2] - pj.v[2] : 0.f};
            float s = w[0] * d[0];
            s = fmaf(w[1], d[1], s);
            if (DIM == 3) s = fmaf(w[2], d[2], s);
            const float invR = fast_rcp(r2 + hc.e2);
            const float u = r2 * invR;
            const float ir_j = 1.0f / pj.rho;
            const float m_j = pj.V * pj.rho;
            const float drho = pi.rho - pj.rho;
            const float W2 = ir_i * ir_j;
            // pressure pair factor e (see k_rhs): form 1 = (p_i + p_j)/(rho_i rho_j) with p = P rho^2
            const float Psum = kp.form == 0 ? pi.P + pj.P : fmaf(pi.P * pi.rho, pi.rho, pj.P * pj.rho * pj.rho) * W2;
            float mm = mu_i[0] * d[0];                          // mu_i . d
            mm = fmaf(mu_i[1], d[1], mm);
            if (DIM == 3) mm = fmaf(mu_i[2], d[2], mm);
            float mmj = mu_j[0] * d[0];                         // mu_j . d   (pair (j<-i) uses -d)
            mmj = fmaf(mu_j[1], d[1], mmj);
            if (DIM == 3) mmj = fmaf(mu_j[2], d[2], mmj);
            const float mmp = -mmj;
            // ---- ordered pair (i <- j)
            const float VjG = pj.V * G;
            const float E = -m_j * Psum;
            const float Phi1 = kp.rho0 * pj.V * s * invR * ir_i;
            const float Phi = hc.eta * Phi1;
            const float sbar = lam_i * pi.rho * VjG + mm * hc.eta * kp.rho0 * VjG * invR * ir_i;
            const float dif = hc.kd * VjG * u;                   // kd V_j (r2/R) G
            const float r2bar = lam_i * hc.kd * VjG * drho * hc.e2 * invR * invR - mm * Phi * G * invR;
            const float Gbar = lam_i * pj.V * (pi.rho * s + hc.kd * drho * u) + mm * (E + Phi);
            // ---- ordered pair (j <- i): d -> -d, w -> -w, s unchanged
            const float ViG = pi.V * G;
            const float Ep = -m_i * Psum;
            const float Phi1p = kp.rho0 * pi.V * s * invR * ir_j;
            const float Phip = hc.eta * Phi1p;
            const float sbarp = lam_j * pj.rho * ViG + mmp * hc.eta * kp.rho0 * ViG * invR * ir_j;
            const float difp = hc.kd * ViG * u;
            const float r2barp = -lam_j * hc.kd * ViG * drho * hc.e2 * invR * invR - mmp * Phip * G * invR;
            const float ADp = ViG * (pj.rho * s - hc.kd * drho * u);          // A' + D'
            const float Gbarp = lam_j * pi.V * (pj.rho * s - hc.kd * drho * u) + mmp * (Ep + Phip);
            // ---- what lands on particle i
            const float cs = sbar + sbarp;
            const float cd = 2.0f * (r2bar + r2barp) + (Gbar + Gbarp) * K;
            const float ce = (E + Phi) * G, cep = (Ep + Phip) * G;
#pragma unroll
            for (int k = 0; k < DIM; ++k) {
                xb[k] += cs * w[k] + cd * d[k] + ce * mu_i[k] - cep * mu_j[k];
                vb[k] = fmaf(cs, d[k], vb[k]);
            }
            rb += lam_i * (VjG * s + dif) - mm * G * Phi * ir_i                 // first role of (i<-j)
                  - lam_j * (ADp * ir_i + difp) - mmp * G * Phip * ir_i;         // second role of (j<-i)
            {
                const float Gzz = G * (m_j * mm + m_i * mmp);
                if (kp.form == 0) {
                    Z = fmaf(Gzz, 1.0f, Z);                         // -dL/dP_i
                } else {
                    Z = fmaf(Gzz, W2, Z);                           // -dL/dp_i
                    Zr = fmaf(Gzz, Psum, Zr);                       // explicit 1/(rho_i rho_j) dependence
                }
            }
            // ---- scalar parameters, ordered pair (i<-j) only (each ordered pair is owned by one row)
            const float D1 = 2.0f * hc.ell * VjG * drho * u;    // D_ij / (delta c0)
            S_D1 = fmaf(lam_i, D1, S_D1);
            const float xphi1 = mm * G * Phi1;
            S_P1 += xphi1;
            S_PL = fmaf(xphi1, hc.ell, S_PL);
            S_eps -= (lam_i * hc.kd * VjG * drho * u + mm * G * Phi) * invR * (2.0f * kp.eps * hc.H2);
        }
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
            xb[k] = group_sum<GS>(xb[k]);
            vb[k] = group_sum<GS>(vb[k]);
        }
        rb = group_sum<GS>(rb);
        Z = group_sum<GS>(Z);
        Zr = group_sum<GS>(Zr);
        if (gl == 0) {
            if (kp.form == 0) {
                rb -= ei.x * Z;                                  // rho_bar_i += Pbar_i dP/drho, Pbar_i = -Z_i
                T_E += pi.P * Z;
                T_0 += ei.y * Z;
                T_g += ei.z * Z;
            } else {
                // form 1: the EOS enters through p = P rho^2: dp/drho = (dP/drho + 2 P/rho) rho^2, dp/dtheta = dP/dtheta rho^2
                const float r2i = pi.rho * pi.rho;
                rb += fmaf(-(ei.x + 2.0f * pi.P * ir_i) * r2i, Z, ir_i * Zr);
                T_E += pi.P * r2i * Z;
                T_0 += ei.y * r2i * Z;
                T_g += ei.z * r2i * Z;
            }
            G0 += mu_i[0]; G1 += mu_i[1]; G2 += mu_i[2];
            if (OUT_SORTED) {
                xb4[row] = make_float4(xb[0], xb[1], xb[2], rb);
                vb4[row] = make_float4(vb[0], vb[1], vb[2], 0.f);
            } else {
                const int64_t i = perm[row];
#pragma unroll
                for (int k = 0; k < DIM; ++k) {
                    xb_out[i * DIM + k] = xb[k];
                    vb_out[i * DIM + k] = vb[k];
                }
                rb_out[i] = rb;
            }
        }
    }
    // B2 stage 1: fixed-order block reduction of the ten partial sums
    __shared__ float red[kBlock / 32][kNPart];
    float vals[10] = {S_D1, S_P1, S_PL, S_eps, T_E, T_0, T_g, G0, G1, G2};
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 10; ++k) {
        float v = vals[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < 10) {
        float v = 0.f;
        for (int w = 0; w < kBlock / 32; ++w) v += red[w][threadIdx.x];
        partials[(int64_t)blockIdx.x * kNPart + threadIdx.x] = v;
    }
}

// ------------------------------------------------------------------------------------------ delta-term of [43], generic lists
// Same sums as k_delta_term_tile (sph_pairs_tile.cu) on the 32-bit sorted-id lists with global gathers.
template <int DIM, int GS, bool VARH, bool ADJ>
__global__ void __launch_bounds__(kBlock)
k_delta_term(int64_t n, KPar kp, float margin, const float4 *__restrict__ pos4, const float4 *__restrict__ g4,
             const float2 *__restrict__ lr, const long long *__restrict__ row_ptr, const int32_t *__restrict__ col,
             const uint32_t *__restrict__ perm, float *__restrict__ drho_io, float4 *__restrict__ out4_io,
             float4 *__restrict__ dx4, float4 *__restrict__ gb4, float *__restrict__ partial)
{
    constexpr int kGroups = kBlock / GS;
    const int g = threadIdx.x / GS, gl = threadIdx.x % GS;
    const int64_t row0 = (int64_t)blockIdx.x * kGroups * kRowsPerGroup;
    const HC hu = hc_uniform<DIM>(kp);
    float SX = 0.f;
    for (int rr = 0; rr < kRowsPerGroup; ++rr) {
        const int64_t row = row0 + (int64_t)rr * kGroups + g;
        if (row >= n) break;
        const float4 pi = __ldg(pos4 + row), gi = __ldg(g4 + row);
        float2 li = make_float2(0.f, 1.f);
        if (ADJ) li = __ldg(lr + row);
        const float xi[3] = {pi.x, pi.y, pi.z};
        const bool seam = row_near_seam(xi, kp, margin);
        const long long b = row_ptr[row], e = row_ptr[row + 1];
        float acc = 0.f, xb[3] = {0.f, 0.f, 0.f}, gb[3] = {0.f, 0.f, 0.f}, rb = 0.f;
        for (long long p = b + gl; p < e; p += GS) {
            const int32_t j = __ldg(col + p);
            const float4 pj = __ldg(pos4 + j), gj = __ldg(g4 + j);
            const float xj[3] = {pj.x, pj.y, pj.z};
            float d[3], r2;
            if (seam) rel_pos<DIM, true>(xi, xj, kp, d, r2); else rel_pos<DIM, false>(xi, xj, kp, d, r2);
            HC hc = hu;
            if (VARH) hc = hc_make<DIM>(fmaxf(pi.w, pj.w), kp);
            const float rr2 = fast_sqrt(r2);
            const float t = fmaxf(fmaf(-hc.invH, rr2, 1.0f), 0.f);
            const float t2 = t * t, t4 = t2 * t2;
            const float G = hc.cG * fmaf(5.0f * hc.invH, rr2, 1.0f) * (t4 * t);
            const float gs[3] = {gi.x + gj.x, gi.y + gj.y, DIM == 3 ? gi.z + gj.z : 0.f};
            const float S = fmaf(gs[2], d[2], fmaf(gs[1], d[1], gs[0] * d[0]));
            const float cc = VARH ? -0.5f * hc.kd : 1.0f;
            if (!ADJ) {
                acc = fmaf(cc * gj.w, S * G, acc);
            } else {
                const float2 lj = __ldg(lr + j);
                const float K = hc.cK * t4;
                const float w = cc * fmaf(li.x, gj.w, -(lj.x * gi.w));
                const float SK = S * K;
#pragma unroll
                for (int kk = 0; kk < DIM; ++kk) {
                    xb[kk] = fmaf(w, fmaf(gs[kk], G, SK * d[kk]), xb[kk]);
                    gb[kk] = fmaf(w * G, d[kk], gb[kk]);
                }
                rb = fmaf(cc * lj.x, S * G, rb);
                SX = fmaf(cc * li.x * gj.w, S * G, SX);
            }
        }
        const float cu = VARH ? 1.0f : -0.5f * hu.kd;
        if (!ADJ) {
            acc = group_sum<GS>(acc) * cu;
            if (gl == 0) {
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
            if (gl == 0) {
                dx4[row] = make_float4(xb[0], xb[1], xb[2], rb);
                gb4[row] = make_float4(gb[0], gb[1], gb[2], 0.f);
            }
        }
    }
    if (ADJ) {
        __shared__ float red[kBlock / 32];
        if (!VARH) SX *= -0.5f * hu.kd;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) SX += __shfl_xor_sync(0xffffffffu, SX, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = SX;
        __syncthreads();
        if (threadIdx.x == 0) {
            float v = 0.f;
            for (int w = 0; w < kBlock / 32; ++w) v += red[w];
            partial[blockIdx.x] = v;
        }
    }
}

// g = M^+ b in sorted order as {g, V} (gbar4 == nullptr), or the records of the adjoint pair pass for a sorted
// cotangent gbar4 (see k_renorm_solve_vjp)
template <int DIM>
__global__ void k_renorm_solve_sorted(int64_t n, const float4 *__restrict__ mom, const float2 *__restrict__ va_s,
                                      const float4 *__restrict__ gbar4, float rcond, float4 *__restrict__ g4_out,
                                      float4 *__restrict__ rb, float4 *__restrict__ rc, float2 *__restrict__ rd,
                                      float *__restrict__ re)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    float m[6], b[3], L[3][3], P[3][3];
    renorm_load<DIM>(mom, p, m, b);
    renorm_pinv<DIM>(m, rcond, L, P);
    float g[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) g[r] = fmaf(L[r][0], b[0], fmaf(L[r][1], b[1], L[r][2] * b[2]));
    const float2 va = va_s[p];
    if (!gbar4) {
        g4_out[p] = make_float4(g[0], g[1], g[2], va.x);
        return;
    }
    const float4 q = gbar4[p];
    const float gb[3] = {q.x, q.y, DIM == 3 ? q.z : 0.f};
    float bb[3], c[3], u[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        bb[r] = fmaf(L[r][0], gb[0], fmaf(L[r][1], gb[1], L[r][2] * gb[2]));
        c[r] = gb[r] - fmaf(P[r][0], gb[0], fmaf(P[r][1], gb[1], P[r][2] * gb[2]));
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) u[r] = fmaf(L[r][0], g[0], fmaf(L[r][1], g[1], L[r][2] * g[2]));
    auto N = [&](int r, int s) { return -(bb[r] * g[s] + g[r] * bb[s]) + (c[r] * u[s] + u[r] * c[s]); };
    rb[p] = make_float4(va.x, va.y, bb[0], bb[1]);
    if (DIM == 3) {
        rc[p] = make_float4(bb[2], N(0, 0), N(0, 1), N(0, 2));
        rd[p] = make_float2(N(1, 1), N(1, 2));
        re[p] = N(2, 2);
    } else {
        rd[p] = make_float2(N(0, 0), N(0, 1));
        re[p] = N(1, 1);
    }
}

// B2 stage 2: one block, binary64 accumulation of the per-block partials in index order, then the chain rule
// from the ten sums to params_bar = d/d{c0, rho0, gamma, delta, alpha, nu, eps, g0, g1, g2}.
constexpr int kReduceThreads = 512;
__global__ void __launch_bounds__(kReduceThreads)
k_reduce_params(int64_t nblocks, const float *__restrict__ partials, KPar kp, int accumulate,
                                float *__restrict__ params_bar)
{
    __shared__ double sh[10][kReduceThreads];
    __shared__ double S[10];
    double acc[10];
    for (int k = 0; k < 10; ++k) acc[k] = 0.0;
    for (int64_t b = threadIdx.x; b < nblocks; b += blockDim.x)
        for (int k = 0; k < 10; ++k) acc[k] += (double)partials[b * kNPart + k];
    for (int k = 0; k < 10; ++k) sh[k][threadIdx.x] = acc[k];
    __syncthreads();
    if (threadIdx.x < 10) {                                  // thread k: sum k over the threads, in index order
        double v = 0.0;
        for (int t = 0; t < (int)blockDim.x; ++t) v += sh[threadIdx.x][t];
        S[threadIdx.x] = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double S_D1 = S[0], S_P1 = S[1], S_PL = S[2], S_eps = S[3], T_E = S[4], T_0 = S[5], T_g = S[6];
        const double c0 = kp.c0, rho0 = kp.rho0, visc = kp.visc_nu;
        double out[10];
        // D = delta c0 D1;  Phi = (alpha l c0 + 2(d+2) nu) Phi1;  P scales with c0^2;  Pbar_i = -Z_i
        out[0] = kp.delta * S_D1 + kp.alpha * S_PL - 2.0 * T_E / c0;                 // c0
        out[1] = (kp.alpha * c0 * S_PL + visc * S_P1) / rho0 - T_0;                  // rho0
        out[2] = -T_g;                                                               // gamma
        out[3] = c0 * S_D1;                                                          // delta
        out[4] = c0 * S_PL;                                                          // alpha
        out[5] = 2.0 * (kp.dim + 2) * S_P1;                                          // nu
        out[6] = S_eps;                                                              // eps
        out[7] = S[7]; out[8] = S[8]; out[9] = S[9];                                 // g
        for (int k = 0; k < 10; ++k) params_bar[k] = (accumulate ? params_bar[k] : 0.f) + (float)out[k];
    }
}

} // namespace

// ==========================================================================================
// host side
// ==========================================================================================
static const double kKappa2 = 2.171239, kKappa3 = 2.207940;

int sph_kpar_make(const sph_ctx *ctx, const sph_params *par, KPar *kp)
{
    if (!(par->c0 > 0.f) || !(par->rho0 > 0.f) || !(par->eps > 0.f) || !(par->gamma > 0.f)) return SPH_E_INVALID;
    if (par->pressure_form != 0 && par->pressure_form != 1) return SPH_E_INVALID;
    if (par->delta_form != 0 && par->delta_form != 1) return SPH_E_INVALID;
    if (par->delta_form == 1 && !(par->renorm_rcond >= 0.f && par->renorm_rcond < 1.f)) return SPH_E_INVALID;
    const GridGeom &gg = ctx->geom;
    memset(kp, 0, sizeof(*kp));
    kp->dim = gg.dim;
    kp->form = par->pressure_form;
    kp->delta_form = par->delta_form;
    kp->rcond = par->renorm_rcond;
    for (int k = 0; k < 3; ++k) {
        kp->periodic[k] = gg.periodic[k];
        kp->L[k] = gg.L[k];
        kp->halfL[k] = 0.5f * gg.L[k];
        kp->lo[k] = gg.lo[k];
        kp->hi[k] = gg.hi[k];
        kp->g[k] = k < gg.dim ? par->g[k] : 0.f;
    }
    kp->c0 = par->c0; kp->rho0 = par->rho0; kp->gamma = par->gamma; kp->delta = par->delta;
    kp->alpha = par->alpha; kp->nu = par->nu; kp->eps = par->eps;
    const double Cd = gg.dim == 2 ? 9.0 / M_PI : 495.0 / (32.0 * M_PI);
    const double kap = gg.dim == 2 ? kKappa2 : kKappa3;
    kp->Cd = (float)Cd;
    kp->inv_kappa = (float)(1.0 / kap);
    kp->visc_nu = (float)(2.0 * (gg.dim + 2) * (double)par->nu);
    kp->Bp = (float)((double)par->rho0 * par->c0 * par->c0 / par->gamma);
    kp->uniform_h = ctx->hmin == ctx->hmax;
    if (kp->uniform_h) {
        const double H = ctx->hmax, iH = 1.0 / H;
        kp->H = (float)H;
        kp->invH = (float)iH;
        kp->cW = (float)(Cd * pow(iH, gg.dim));
        kp->cG = (float)(-(56.0 / 3.0) * Cd * pow(iH, gg.dim + 2));
        kp->cK = (float)(560.0 * Cd * pow(iH, gg.dim + 4));
        const double ell = H / kap;
        kp->ell = (float)ell;
        kp->e2 = (float)((par->eps * H) * (par->eps * H));
        kp->eta = (float)((double)par->alpha * ell * par->c0 + 2.0 * (gg.dim + 2) * (double)par->nu);
        kp->kd = (float)(2.0 * (double)par->delta * ell * par->c0);
    }
    return SPH_OK;
}

namespace {

// margin of row_near_seam: the list radius plus the largest admissible drift of a skin list
float seam_margin(const sph_ctx *ctx)
{
    double e = 0.0;
    for (int k = 0; k < ctx->geom.dim; ++k)
        if (ctx->geom.edge[k] > e) e = ctx->geom.edge[k];
    return (float)(2.0 * e);
}

unsigned pair_grid(int64_t n, int gs) { return (unsigned)((n + (kBlock / gs) * kRowsPerGroup - 1) / ((kBlock / gs) * kRowsPerGroup)); }

template <int DIM>
int pack_state(sph_ctx *ctx, const KPar &kp, const float *x, const float *v, const float *rho, const float *m,
               const uint8_t *kind, bool with_eos, cudaStream_t st)
{
    const int64_t n = ctx->n;
    SPH_TRY(ctx->s0.reserve((size_t)n * 16));
    SPH_TRY(ctx->s1.reserve((size_t)n * 16));
    SPH_TRY(ctx->s2.reserve((size_t)n * 8));
    SPH_TRY(ctx->kind_s.reserve((size_t)n));
    if (with_eos) SPH_TRY(ctx->eos.reserve((size_t)n * 16));
    KScope ks(ctx, SPH_K_PACK, 1, st);
    SPH_CUDA_TRY(cudaMemsetAsync(sph_um_flag(ctx), 1, 4, st));       // "masses uniform" until a thread finds otherwise
    k_pack_state<DIM><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(
        n, kp, ctx->perm.as<uint32_t>(), ctx->pos_s.as<float4>(), x, v, rho, m, kind, ctx->s0.as<float4>(),
        ctx->s1.as<float4>(), ctx->s2.as<float2>(), with_eos ? ctx->eos.as<float4>() : nullptr, ctx->kind_s.as<uint8_t>(),
        sph_um_flag(ctx));
    return SPH_OK;
}

} // namespace

// sorted-state launchers (also used by sph_rk.cu)
int sph_launch_rhs_sorted(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                          const uint8_t *kind_s, float *drho, float *acc, float4 *out4, cudaStream_t st)
{
    const int64_t n = ctx->n;
    const float margin = seam_margin(ctx);
    const long long *rp = ctx->row_ptr.as<long long>();
    const int32_t *col = ctx->col.as<int32_t>();
    const uint32_t *perm = ctx->perm.as<uint32_t>();
    const bool sorted = out4 != nullptr;
    if (ctx->tile_mode) {
        {
            KScope ks(ctx, SPH_K_RHS, 1, st);
            SPH_TRY(sph_launch_rhs_tile(ctx, kp, s0, s1, s2, kind_s, drho, acc, out4, st));
        }
        if (kp.delta_form == 1) SPH_TRY(sph_delta_forward(ctx, kp, s0, s1, s2, drho, out4, st));
        return SPH_OK;
    }
    {
    KScope ks(ctx, SPH_K_RHS, 1, st);
#define SPH_RHS_LAUNCH(DIM, GS, VARH, SORTED)                                                                     \
    k_rhs<DIM, GS, VARH, SORTED><<<pair_grid(n, GS), kBlock, 0, st>>>(n, kp, margin, s0, s1, s2, kind_s, rp, col, \
                                                                     perm, drho, acc, out4)
#define SPH_RHS_GS(GS)                                                                                              \
    if (kp.dim == 3) {                                                                                              \
        if (kp.uniform_h) { if (sorted) SPH_RHS_LAUNCH(3, GS, false, true); else SPH_RHS_LAUNCH(3, GS, false, false); } \
        else { if (sorted) SPH_RHS_LAUNCH(3, GS, true, true); else SPH_RHS_LAUNCH(3, GS, true, false); }                \
    } else {                                                                                                        \
        if (kp.uniform_h) { if (sorted) SPH_RHS_LAUNCH(2, GS, false, true); else SPH_RHS_LAUNCH(2, GS, false, false); } \
        else { if (sorted) SPH_RHS_LAUNCH(2, GS, true, true); else SPH_RHS_LAUNCH(2, GS, true, false); }                \
    }
    const int gs_ = ctx->opt_group ? ctx->opt_group : (kp.dim == 3 ? 32 : 16);
    switch (gs_) {
    case 4: SPH_RHS_GS(4) break;
    case 8: SPH_RHS_GS(8) break;
    case 16: SPH_RHS_GS(16) break;
    default: SPH_RHS_GS(32) break;
    }
#undef SPH_RHS_GS
#undef SPH_RHS_LAUNCH
    }
    SPH_CUDA_TRY(cudaGetLastError());
    if (kp.delta_form == 1) SPH_TRY(sph_delta_forward(ctx, kp, s0, s1, s2, drho, out4, st));
    return SPH_OK;
}

int sph_launch_vjp_sorted(sph_ctx *ctx, const KPar &kp, const float4 *s0, const float4 *s1, const float2 *s2,
                          const float4 *cot, const float4 *eos, float *xb, float *vb, float *rb, float4 *xb4,
                          float4 *vb4, float *params_bar, int accumulate_params, cudaStream_t st)
{
    const int64_t n = ctx->n;
    const float margin = seam_margin(ctx);
    const long long *rp = ctx->row_ptr.as<long long>();
    const int32_t *col = ctx->col.as<int32_t>();
    const uint32_t *perm = ctx->perm.as<uint32_t>();
    const bool sorted = xb4 != nullptr;
    const int gs = ctx->opt_group ? ctx->opt_group : (kp.dim == 3 ? 32 : 16);
    const unsigned grid = ctx->tile_mode ? (unsigned)ctx->tg.ntiles * (unsigned)sph_vjp_tile_split(ctx, kp) : pair_grid(n, gs);
    SPH_TRY(ctx->partials.reserve((size_t)grid * kNPart * 4));
    float *part = ctx->partials.as<float>();
    if (ctx->tile_mode) {
        KScope ks(ctx, SPH_K_VJP, 1, st);
        SPH_TRY(sph_launch_vjp_tile(ctx, kp, s0, s1, s2, cot, eos, xb, vb, rb, xb4, vb4, part, st));
    } else {
    KScope ks(ctx, SPH_K_VJP, 1, st);
#define SPH_VJP_LAUNCH(DIM, GS, VARH, SORTED)                                                                  \
    k_vjp<DIM, GS, VARH, SORTED><<<grid, kBlock, 0, st>>>(n, kp, margin, s0, s1, s2, cot, eos, rp, col, perm, xb, \
                                                         vb, rb, xb4, vb4, part)
#define SPH_VJP_GS(GS)                                                                                              \
    if (kp.dim == 3) {                                                                                              \
        if (kp.uniform_h) { if (sorted) SPH_VJP_LAUNCH(3, GS, false, true); else SPH_VJP_LAUNCH(3, GS, false, false); } \
        else { if (sorted) SPH_VJP_LAUNCH(3, GS, true, true); else SPH_VJP_LAUNCH(3, GS, true, false); }                \
    } else {                                                                                                        \
        if (kp.uniform_h) { if (sorted) SPH_VJP_LAUNCH(2, GS, false, true); else SPH_VJP_LAUNCH(2, GS, false, false); } \
        else { if (sorted) SPH_VJP_LAUNCH(2, GS, true, true); else SPH_VJP_LAUNCH(2, GS, true, false); }                \
    }
    switch (gs) {
    case 4: SPH_VJP_GS(4) break;
    case 8: SPH_VJP_GS(8) break;
    case 16: SPH_VJP_GS(16) break;
    default: SPH_VJP_GS(32) break;
    }
#undef SPH_VJP_GS
#undef SPH_VJP_LAUNCH
    }
    if (params_bar) {
        KScope ks(ctx, SPH_K_REDUCE, 1, st);
        k_reduce_params<<<1, kReduceThreads, 0, st>>>((int64_t)grid, part, kp, accumulate_params, params_bar);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    if (kp.delta_form == 1) SPH_TRY(sph_delta_adjoint(ctx, kp, s0, s1, s2, cot, xb, rb, xb4, params_bar, st));
    return SPH_OK;
}

int sph_delta_term_generic(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *g4, const float2 *lr, bool adjoint,
                           float *drho_io, float4 *out4_io, float4 *dx4, float4 *gb4, float *partial, int *npartial,
                           cudaStream_t st)
{
    const int64_t n = ctx->n;
    const float margin = seam_margin(ctx);
    const int gs = kp.dim == 3 ? 32 : 16;
    const unsigned grid = pair_grid(n, gs);
    if (npartial) *npartial = (int)grid;
#define SPH_DG_LAUNCH(DIM, GS, VARH, ADJ)                                                                          \
    k_delta_term<DIM, GS, VARH, ADJ><<<grid, kBlock, 0, st>>>(n, kp, margin, pos4, g4, lr, ctx->row_ptr.as<long long>(), \
                                                             ctx->col.as<int32_t>(), ctx->perm.as<uint32_t>(), drho_io,  \
                                                             out4_io, dx4, gb4, partial)
    if (kp.dim == 3) {
        if (kp.uniform_h) { if (adjoint) SPH_DG_LAUNCH(3, 32, false, true); else SPH_DG_LAUNCH(3, 32, false, false); }
        else { if (adjoint) SPH_DG_LAUNCH(3, 32, true, true); else SPH_DG_LAUNCH(3, 32, true, false); }
    } else {
        if (kp.uniform_h) { if (adjoint) SPH_DG_LAUNCH(2, 16, false, true); else SPH_DG_LAUNCH(2, 16, false, false); }
        else { if (adjoint) SPH_DG_LAUNCH(2, 16, true, true); else SPH_DG_LAUNCH(2, 16, true, false); }
    }
#undef SPH_DG_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int sph_renorm_solve_sorted(sph_ctx *ctx, const KPar &kp, const float4 *mom, const float2 *va_s, const float4 *gbar4,
                            float4 *g4_out, float4 *rb, float4 *rc, float2 *rd, float *re, cudaStream_t st)
{
    const int64_t n = ctx->n;
    const unsigned nb1 = (unsigned)((n + 255) / 256);
    if (kp.dim == 3) k_renorm_solve_sorted<3><<<nb1, 256, 0, st>>>(n, mom, va_s, gbar4, kp.rcond, g4_out, rb, rc, rd, re);
    else k_renorm_solve_sorted<2><<<nb1, 256, 0, st>>>(n, mom, va_s, gbar4, kp.rcond, g4_out, rb, rc, rd, re);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_density(sph_ctx *ctx, const float *m, float *rho_out, sph_stream_t stream)
{
    if (!ctx || !m || !rho_out) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    sph_params dummy{};
    dummy.c0 = 1.f; dummy.rho0 = 1.f; dummy.gamma = 1.f; dummy.eps = 1.f;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, &dummy, &kp));
    SPH_TRY(ctx->m_s.reserve((size_t)n * 4));
    KScope ks(ctx, SPH_K_DENSITY, 2, st);
    if (ctx->tile_mode) {
        // uniform-mass fast path (SPH_OPT_UNIFORM_MASS_PATH): the gather kernel leaves "all masses equal" in a device flag
        uint32_t *um = ctx->opt_no_um ? nullptr : ctx->stats.as<uint32_t>() + kDensUmSlot;
        if (um) {
            SPH_CUDA_TRY(cudaMemsetAsync(um, 1, 4, st));
            k_gather_f32_um<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), m, ctx->m_s.as<float>(), um);
        } else {
            k_gather_f32<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), m, ctx->m_s.as<float>());
        }
        return sph_launch_density_tile(ctx, kp, ctx->m_s.as<float>(), rho_out, um, m, st);
    }
    k_gather_f32<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), m, ctx->m_s.as<float>());
    const float margin = seam_margin(ctx);
#define SPH_DENS_LAUNCH(DIM, GS, VARH)                                                                               \
    k_density<DIM, GS, VARH><<<pair_grid(n, GS), kBlock, 0, st>>>(n, kp, margin, ctx->pos_s.as<float4>(),           \
                                                                 ctx->m_s.as<float>(), ctx->row_ptr.as<long long>(), \
                                                                 ctx->col.as<int32_t>(), ctx->perm.as<uint32_t>(), rho_out)
    if (kp.dim == 3) { if (kp.uniform_h) SPH_DENS_LAUNCH(3, 32, false); else SPH_DENS_LAUNCH(3, 32, true); }
    else { if (kp.uniform_h) SPH_DENS_LAUNCH(2, 16, false); else SPH_DENS_LAUNCH(2, 16, true); }
#undef SPH_DENS_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_density_vjp(sph_ctx *ctx, const float *m, const float *rho_bar, float *x_bar, float *m_bar,
                               sph_stream_t stream)
{
    if (!ctx || !m || !rho_bar || !x_bar) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    sph_params dummy{};
    dummy.c0 = 1.f; dummy.rho0 = 1.f; dummy.gamma = 1.f; dummy.eps = 1.f;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, &dummy, &kp));
    SPH_TRY(ctx->s2.reserve((size_t)n * 8));
    float2 *mr_s = ctx->s2.as<float2>();
    KScope ks(ctx, SPH_K_DENSITY, 2, st);
    k_gather_f32x2<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), m, rho_bar, mr_s);
    if (ctx->tile_mode) return sph_launch_density_vjp_tile(ctx, kp, mr_s, x_bar, m_bar, st);
    const float margin = seam_margin(ctx);
#define SPH_DVJP_LAUNCH(DIM, GS, VARH)                                                                                 \
    k_density_vjp<DIM, GS, VARH><<<pair_grid(n, GS), kBlock, 0, st>>>(n, kp, margin, ctx->pos_s.as<float4>(), mr_s,    \
                                                                     ctx->row_ptr.as<long long>(), ctx->col.as<int32_t>(), \
                                                                     ctx->perm.as<uint32_t>(), x_bar, m_bar)
    if (kp.dim == 3) { if (kp.uniform_h) SPH_DVJP_LAUNCH(3, 32, false); else SPH_DVJP_LAUNCH(3, 32, true); }
    else { if (kp.uniform_h) SPH_DVJP_LAUNCH(2, 16, false); else SPH_DVJP_LAUNCH(2, 16, true); }
#undef SPH_DVJP_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

static int grad_sum_common(sph_ctx *ctx, const float *a, const float *g_bar, float *v_out, float *a_out, bool vjp,
                           cudaStream_t st)
{
    const int64_t n = ctx->n;
    sph_params dummy{};
    dummy.c0 = 1.f; dummy.rho0 = 1.f; dummy.gamma = 1.f; dummy.eps = 1.f;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, &dummy, &kp));
    KScope ks(ctx, SPH_K_DENSITY, 2, st);
    const unsigned nb1 = (unsigned)((n + 255) / 256);
    if (!vjp && ctx->tile_mode) {
        SPH_TRY(ctx->m_s.reserve((size_t)n * 4));
        k_gather_f32<<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), a, ctx->m_s.as<float>());
        return sph_launch_grad_sum_tile(ctx, kp, ctx->m_s.as<float>(), v_out, st);
    }
    SPH_TRY(ctx->c0buf.reserve((size_t)n * 16));
    float4 *ga = ctx->c0buf.as<float4>();
    // forward on the generic layout: the weights ride in .w of the same float4 record (xyz unused)
    const float *vec = vjp ? g_bar : nullptr;
    if (kp.dim == 3) {
        if (vec) k_gather_vec_a<3><<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), vec, a, ga);
        else k_gather_f32_w<<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), a, ga);
    } else {
        if (vec) k_gather_vec_a<2><<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), vec, a, ga);
        else k_gather_f32_w<<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), a, ga);
    }
    if (ctx->tile_mode) return sph_launch_grad_sum_vjp_tile(ctx, kp, ga, v_out, a_out, st);
    const float margin = seam_margin(ctx);
#define SPH_GS_LAUNCH(DIM, GS, VARH, VJP)                                                                             \
    k_grad_sum<DIM, GS, VARH, VJP><<<pair_grid(n, GS), kBlock, 0, st>>>(n, kp, margin,                                \
                                                                       ctx->pos_override ? ctx->pos_override : ctx->pos_s.as<float4>(), ga, \
                                                                       ctx->row_ptr.as<long long>(), ctx->col.as<int32_t>(), \
                                                                       ctx->perm.as<uint32_t>(), v_out, a_out)
#define SPH_GS_DIM(DIM, GS)                                                                                  \
    do {                                                                                                     \
        if (kp.uniform_h) { if (vjp) SPH_GS_LAUNCH(DIM, GS, false, true); else SPH_GS_LAUNCH(DIM, GS, false, false); } \
        else { if (vjp) SPH_GS_LAUNCH(DIM, GS, true, true); else SPH_GS_LAUNCH(DIM, GS, true, false); }               \
    } while (0)
    if (kp.dim == 3) SPH_GS_DIM(3, 32); else SPH_GS_DIM(2, 16);
#undef SPH_GS_DIM
#undef SPH_GS_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_grad_sum(sph_ctx *ctx, const float *a, float *g_out, sph_stream_t stream)
{
    if (!ctx || !a || !g_out) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    ctx->last_stream = (cudaStream_t)stream;
    return grad_sum_common(ctx, a, nullptr, g_out, nullptr, false, (cudaStream_t)stream);
}

extern "C" int sph_grad_sum_vjp(sph_ctx *ctx, const float *a, const float *g_bar, float *x_bar, float *a_bar,
                                sph_stream_t stream)
{
    if (!ctx || !a || !g_bar || !x_bar) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    ctx->last_stream = (cudaStream_t)stream;
    return grad_sum_common(ctx, a, g_bar, x_bar, a_bar, true, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------ particle shifting
// End-of-step particle shifting ("particle-shifting only at the end of each overall timestep", PAPER.md:680;
// the scheme of [41] is not printed -- DESIGN.md reading R18: the Fickian form, shift along the gradient of the particle
// concentration C_i = sum_j V_j W_ij):   x_i <- x_i - theta l_i^2 sum_j V_j grad_i W_ij   for fluid kinds, l = h/kappa_d.
// The sum is sph_grad_sum with a = m/rho, evaluated at the CURRENT positions on the lists of the last build (valid as
// long as they are a superset of the neighbours, e.g. right after sph_rk_step with its skin).
namespace {
template <int DIM>
__global__ void k_shift_prep(int64_t n, KPar kp, const uint32_t *__restrict__ perm, const float4 *__restrict__ pos_s,
                             const float *__restrict__ x, const float *__restrict__ m, const float *__restrict__ rho,
                             float4 *__restrict__ pos4, float *__restrict__ vol)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int64_t i = perm[p];
    const float4 pb = pos_s[p];
    const float xb[3] = {pb.x, pb.y, pb.z};
    float xw[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        float xv = x[i * DIM + k];
        if (kp.periodic[k]) {                                  // the periodic image next to the build position (k_pack_state)
            xv = wrap_coord(xv, kp.lo[k], kp.hi[k], kp.L[k]);
            const float dd = xv - xb[k];
            xv = dd > kp.halfL[k] ? xv - kp.L[k] : (dd < -kp.halfL[k] ? xv + kp.L[k] : xv);
        }
        xw[k] = xv;
    }
    pos4[p] = make_float4(xw[0], xw[1], xw[2], pb.w);
    vol[i] = m[i] / rho[i];                                    // caller order: the weights of sph_grad_sum
}
template <int DIM>
__global__ void k_shift_apply(int64_t n, float theta, float inv_kappa, const uint32_t *__restrict__ inv_perm,
                              const float4 *__restrict__ pos_s, const uint8_t *__restrict__ kind, const float *__restrict__ g,
                              float *__restrict__ x)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || kind[i]) return;
    const float ell = pos_s[inv_perm[i]].w * inv_kappa;
    const float c = -theta * ell * ell;
#pragma unroll
    for (int k = 0; k < DIM; ++k) x[i * DIM + k] = fmaf(c, g[i * DIM + k], x[i * DIM + k]);
}
} // namespace

extern "C" int sph_shift(sph_ctx *ctx, float theta, float *x, const float *m, const float *rho, const uint8_t *kind,
                         sph_stream_t stream)
{
    if (!ctx || !x || !m || !rho || !kind || !isfinite(theta)) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    sph_params dummy{};
    dummy.c0 = 1.f; dummy.rho0 = 1.f; dummy.gamma = 1.f; dummy.eps = 1.f;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, &dummy, &kp));
    SPH_TRY(ctx->d_pos.reserve((size_t)n * 16));
    SPH_TRY(ctx->d_vb.reserve((size_t)n * 4));
    SPH_TRY(ctx->d_x2.reserve((size_t)n * 12));
    const unsigned nb1 = (unsigned)((n + 255) / 256);
    {
        KScope ks(ctx, SPH_K_PACK, 1, st);
        if (kp.dim == 3) k_shift_prep<3><<<nb1, 256, 0, st>>>(n, kp, ctx->perm.as<uint32_t>(), ctx->pos_s.as<float4>(), x, m, rho, ctx->d_pos.as<float4>(), ctx->d_vb.as<float>());
        else k_shift_prep<2><<<nb1, 256, 0, st>>>(n, kp, ctx->perm.as<uint32_t>(), ctx->pos_s.as<float4>(), x, m, rho, ctx->d_pos.as<float4>(), ctx->d_vb.as<float>());
    }
    ctx->pos_override = ctx->d_pos.as<float4>();
    const int rc = grad_sum_common(ctx, ctx->d_vb.as<float>(), nullptr, ctx->d_x2.as<float>(), nullptr, false, st);
    ctx->pos_override = nullptr;
    SPH_TRY(rc);
    {
        KScope ks(ctx, SPH_K_RK, 1, st);
        if (kp.dim == 3) k_shift_apply<3><<<nb1, 256, 0, st>>>(n, theta, kp.inv_kappa, ctx->inv_perm.as<uint32_t>(), ctx->pos_s.as<float4>(), kind, ctx->d_x2.as<float>(), x);
        else k_shift_apply<2><<<nb1, 256, 0, st>>>(n, theta, kp.inv_kappa, ctx->inv_perm.as<uint32_t>(), ctx->pos_s.as<float4>(), kind, ctx->d_x2.as<float>(), x);
    }
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

// moments M_i, b_i of the kernel renormalisation on either list layout (forward, and recomputed by the adjoint)
int sph_renorm_moments_any(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float2 *va_s, float4 *mom, cudaStream_t st)
{
    if (ctx->tile_mode) return sph_launch_renorm_tile(ctx, kp, pos4, va_s, mom, st);
    const int64_t n = ctx->n;
    const float margin = seam_margin(ctx);
#define SPH_RN_LAUNCH(DIM, GS, VARH)                                                                             \
    k_renorm<DIM, GS, VARH><<<pair_grid(n, GS), kBlock, 0, st>>>(n, kp, margin, pos4, va_s,                      \
                                                                ctx->row_ptr.as<long long>(), ctx->col.as<int32_t>(), mom)
    if (kp.dim == 3) { if (kp.uniform_h) SPH_RN_LAUNCH(3, 32, false); else SPH_RN_LAUNCH(3, 32, true); }
    else { if (kp.uniform_h) SPH_RN_LAUNCH(2, 16, false); else SPH_RN_LAUNCH(2, 16, true); }
#undef SPH_RN_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}
static int launch_renorm_moments(sph_ctx *ctx, const KPar &kp, const float2 *va_s, float4 *mom, cudaStream_t st)
{
    return sph_renorm_moments_any(ctx, kp, ctx->pos_s.as<float4>(), va_s, mom, st);
}

// pair pass of the renormalised-gradient adjoint on given positions; perm == nullptr: outputs in sorted order
int sph_renorm_vjp_pairs_any(sph_ctx *ctx, const KPar &kp, const float4 *pos4, const float4 *rb, const float4 *rc,
                             const float2 *rd, const float *re, const uint32_t *perm, float *x_bar, float *vol_bar,
                             float *A_bar, cudaStream_t st)
{
    if (ctx->tile_mode) return sph_launch_renorm_vjp_tile(ctx, kp, pos4, rb, rc, rd, re, perm, x_bar, vol_bar, A_bar, st);
    const int64_t n = ctx->n;
    const float margin = seam_margin(ctx);
#define SPH_RNV_LAUNCH(DIM, GS, VARH)                                                                                  \
    k_renorm_vjp<DIM, GS, VARH><<<pair_grid(n, GS), kBlock, 0, st>>>(n, kp, margin, pos4, rb, rc, rd,                  \
                                                                    re, ctx->row_ptr.as<long long>(),                   \
                                                                    ctx->col.as<int32_t>(), perm, x_bar, vol_bar, A_bar)
    if (kp.dim == 3) { if (kp.uniform_h) SPH_RNV_LAUNCH(3, 16, false); else SPH_RNV_LAUNCH(3, 16, true); }
    else { if (kp.uniform_h) SPH_RNV_LAUNCH(2, 16, false); else SPH_RNV_LAUNCH(2, 16, true); }
#undef SPH_RNV_LAUNCH
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_renorm_gradient(sph_ctx *ctx, const float *vol, const float *A, float rcond, float *L_out,
                                   float *grad_out, sph_stream_t stream)
{
    if (!ctx || !vol || !A || (!L_out && !grad_out) || !(rcond >= 0.f) || !(rcond < 1.f)) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    sph_params dummy{};
    dummy.c0 = 1.f; dummy.rho0 = 1.f; dummy.gamma = 1.f; dummy.eps = 1.f;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, &dummy, &kp));
    SPH_TRY(ctx->s2.reserve((size_t)n * 8));
    SPH_TRY(ctx->c0buf.reserve((size_t)n * 48));
    float2 *va_s = ctx->s2.as<float2>();
    float4 *mom = ctx->c0buf.as<float4>();
    KScope ks(ctx, SPH_K_DENSITY, 3, st);
    const unsigned nb1 = (unsigned)((n + 255) / 256);
    k_gather_f32x2<<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), vol, A, va_s);
    SPH_TRY(launch_renorm_moments(ctx, kp, va_s, mom, st));
    if (kp.dim == 3) k_renorm_solve<3><<<nb1, 256, 0, st>>>(n, mom, ctx->perm.as<uint32_t>(), rcond, L_out, grad_out);
    else k_renorm_solve<2><<<nb1, 256, 0, st>>>(n, mom, ctx->perm.as<uint32_t>(), rcond, L_out, grad_out);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

extern "C" int sph_renorm_gradient_vjp(sph_ctx *ctx, const float *vol, const float *A, float rcond, const float *grad_bar,
                                       float *x_bar, float *vol_bar, float *A_bar, sph_stream_t stream)
{
    if (!ctx || !vol || !A || !grad_bar || !x_bar || !(rcond >= 0.f) || !(rcond < 1.f)) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    sph_params dummy{};
    dummy.c0 = 1.f; dummy.rho0 = 1.f; dummy.gamma = 1.f; dummy.eps = 1.f;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, &dummy, &kp));
    SPH_TRY(ctx->s2.reserve((size_t)n * 8));
    SPH_TRY(ctx->c0buf.reserve((size_t)n * 48));
    SPH_TRY(ctx->s0.reserve((size_t)n * 16));
    SPH_TRY(ctx->s1.reserve((size_t)n * 16));
    SPH_TRY(ctx->out4.reserve((size_t)n * 16));
    SPH_TRY(ctx->m_s.reserve((size_t)n * 4));
    float2 *va_s = ctx->s2.as<float2>();
    float4 *mom = ctx->c0buf.as<float4>();
    float4 *rb = ctx->s0.as<float4>(), *rc = ctx->s1.as<float4>();
    float2 *rd = ctx->out4.as<float2>();
    float *re = ctx->m_s.as<float>();
    KScope ks(ctx, SPH_K_DENSITY, 4, st);
    const unsigned nb1 = (unsigned)((n + 255) / 256);
    // forward moments again (nothing is kept between calls), then the per-particle adjoint of g = M^+ b
    k_gather_f32x2<<<nb1, 256, 0, st>>>(n, ctx->perm.as<uint32_t>(), vol, A, va_s);
    SPH_TRY(launch_renorm_moments(ctx, kp, va_s, mom, st));
    if (kp.dim == 3)
        k_renorm_solve_vjp<3><<<nb1, 256, 0, st>>>(n, mom, va_s, ctx->perm.as<uint32_t>(), grad_bar, rcond, rb, rc, rd, re);
    else
        k_renorm_solve_vjp<2><<<nb1, 256, 0, st>>>(n, mom, va_s, ctx->perm.as<uint32_t>(), grad_bar, rcond, rb, rc, rd, re);
    return sph_renorm_vjp_pairs_any(ctx, kp, ctx->pos_s.as<float4>(), rb, rc, rd, re, ctx->perm.as<uint32_t>(), x_bar,
                                    vol_bar, A_bar, st);
}

extern "C" int sph_rhs(sph_ctx *ctx, const sph_params *par, const float *x, const float *v, const float *rho,
                       const float *m, const uint8_t *kind, float *drho_dt, float *acc, sph_stream_t stream)
{
    if (!ctx || !par || !x || !v || !rho || !m || !kind || !drho_dt || !acc) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, par, &kp));
    if (kp.dim == 3) SPH_TRY(pack_state<3>(ctx, kp, x, v, rho, m, kind, false, st));
    else SPH_TRY(pack_state<2>(ctx, kp, x, v, rho, m, kind, false, st));
    return sph_launch_rhs_sorted(ctx, kp, ctx->s0.as<float4>(), ctx->s1.as<float4>(), ctx->s2.as<float2>(),
                                 ctx->kind_s.as<uint8_t>(), drho_dt, acc, nullptr, st);
}

extern "C" int sph_rhs_vjp(sph_ctx *ctx, const sph_params *par, const float *x, const float *v, const float *rho,
                           const float *m, const uint8_t *kind, const float *drho_bar, const float *acc_bar,
                           float *x_bar, float *v_bar, float *rho_bar, float *params_bar, sph_stream_t stream)
{
    if (!ctx || !par || !x || !v || !rho || !m || !kind || !drho_bar || !acc_bar || !x_bar || !v_bar || !rho_bar)
        return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    ctx->last_stream = st;
    const int64_t n = ctx->n;
    KPar kp;
    SPH_TRY(sph_kpar_make(ctx, par, &kp));
    if (kp.dim == 3) SPH_TRY(pack_state<3>(ctx, kp, x, v, rho, m, kind, true, st));
    else SPH_TRY(pack_state<2>(ctx, kp, x, v, rho, m, kind, true, st));
    SPH_TRY(ctx->c0buf.reserve((size_t)n * 16));
    {
        KScope ks(ctx, SPH_K_PACK, 1, st);
        k_pack_cot<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, kp.dim, ctx->perm.as<uint32_t>(), ctx->kind_s.as<uint8_t>(),
                                                                drho_bar, acc_bar, ctx->c0buf.as<float4>());
    }
    return sph_launch_vjp_sorted(ctx, kp, ctx->s0.as<float4>(), ctx->s1.as<float4>(), ctx->s2.as<float2>(),
                                 ctx->c0buf.as<float4>(), ctx->eos.as<float4>(), x_bar, v_bar, rho_bar, nullptr, nullptr,
                                 params_bar, 0, st);
}
