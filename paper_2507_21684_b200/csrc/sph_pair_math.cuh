// sph_pair_math.cuh -- H-dependent constants of the Wendland C4 pair terms (Eq.25-29), shared by the
// global-gather pair kernels (sph_pairs.cu) and the tile kernels (sph_pairs_tile.cu).
#pragma once

#include "sph_internal.cuh"

// H-dependent constants of one pair (or of the whole launch when h is uniform)
struct HC {
    float invH, cW, cG, cK, ell, e2, eta, kd, H2;
};

template <int DIM>
static __device__ __forceinline__ HC hc_make(float H, const KPar &kp)
{
    HC c;
    c.invH = 1.0f / H;
    float i2 = c.invH * c.invH;
    float iD = DIM == 2 ? i2 : i2 * c.invH;             // H^-d
    c.cW = kp.Cd * iD;
    c.cG = -(56.0f / 3.0f) * kp.Cd * iD * i2;           // G = cG (1+5q)(1-q)^5
    c.cK = 560.0f * kp.Cd * iD * i2 * i2;               // K = cK (1-q)^4
    c.ell = H * kp.inv_kappa;
    float eh = kp.eps * H;
    c.e2 = eh * eh;
    c.eta = kp.alpha * c.ell * kp.c0 + kp.visc_nu;
    c.kd = 2.0f * kp.delta * c.ell * kp.c0;
    c.H2 = H * H;
    return c;
}
template <int DIM>
static __device__ __forceinline__ HC hc_uniform(const KPar &kp)
{
    HC c;
    c.invH = kp.invH; c.cW = kp.cW; c.cG = kp.cG; c.cK = kp.cK; c.ell = kp.ell; c.e2 = kp.e2; c.eta = kp.eta;
    c.kd = kp.kd; c.H2 = kp.H * kp.H;
    return c;
}

