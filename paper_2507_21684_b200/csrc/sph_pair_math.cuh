// sph_pair_math.cuh -- particle record and H-dependent constants of the Wendland C4 pair terms (Eq.25-29), shared by the
// global-gather pair kernels (sph_pairs.cu) and the tile kernels (sph_pairs_tile.cu).
#pragma once

#include "sph_internal.cuh"

// Sorted state of one particle as the pair loops see it, and the record layout both kernel families read it from:
// DIM 3: s0 = {x,y,z,rho}  s1 = {vx,vy,vz,P}  s2 (float2) = {V,h};   DIM 2: s0 = {x,y,vx,vy}  s1 = {rho,V,P,h}.
// In 3D everything a pair needs when mass and h are uniform sits in s0, s1 (the uniform-mass tile kernels leave s2 out
// and pass V = m0 / rho, h = H instead).
struct Part {
    float x[3], v[3], rho, V, P, h;
};
template <int DIM>
static __device__ __forceinline__ Part part_unpack(const float4 &a, const float4 &b, float V3 = 0.f, float h3 = 0.f)
{
    Part p;
    if (DIM == 3) {
        p.x[0] = a.x; p.x[1] = a.y; p.x[2] = a.z; p.rho = a.w;
        p.v[0] = b.x; p.v[1] = b.y; p.v[2] = b.z; p.P = b.w;
        p.V = V3; p.h = h3;
    } else {
        p.x[0] = a.x; p.x[1] = a.y; p.x[2] = 0.f; p.v[0] = a.z; p.v[1] = a.w; p.v[2] = 0.f;
        p.rho = b.x; p.V = b.y; p.P = b.z; p.h = b.w;
    }
    return p;
}

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

// ------------------------------------------------------------------------------------------ kernel renormalisation, adjoint
// per-particle record of the pair pass of sph_renorm_gradient_vjp (written by k_renorm_solve_vjp, sph_pairs.cu)
struct RenormRec {
    float V, A, bb[3], N[6];                                   // N = {xx, xy, xz, yy, yz, zz}
};
template <int DIM>
static __device__ __forceinline__ RenormRec renorm_rec(const float4 &b, const float4 &c, const float2 &d, float e)
{
    RenormRec r;
    r.V = b.x; r.A = b.y; r.bb[0] = b.z; r.bb[1] = b.w;
    if (DIM == 3) {
        r.bb[2] = c.x; r.N[0] = c.y; r.N[1] = c.z; r.N[2] = c.w; r.N[3] = d.x; r.N[4] = d.y; r.N[5] = e;
    } else {
        r.bb[2] = 0.f; r.N[0] = d.x; r.N[1] = d.y; r.N[2] = 0.f; r.N[3] = e; r.N[4] = 0.f; r.N[5] = 0.f;
    }
    return r;
}
// contributions of neighbour j to row i; d = x_i - x_j
template <int DIM>
static __device__ __forceinline__ void renorm_vjp_pair(const RenormRec &ri, const RenormRec &rj, const float (&d)[3], float G,
                                                float K, float (&xb)[3], float &vb, float &ab)
{
    float Nid[3], Njd[3];
    Nid[0] = fmaf(ri.N[0], d[0], fmaf(ri.N[1], d[1], ri.N[2] * d[2]));
    Nid[1] = fmaf(ri.N[1], d[0], fmaf(ri.N[3], d[1], ri.N[4] * d[2]));
    Nid[2] = fmaf(ri.N[2], d[0], fmaf(ri.N[4], d[1], ri.N[5] * d[2]));
    Njd[0] = fmaf(rj.N[0], d[0], fmaf(rj.N[1], d[1], rj.N[2] * d[2]));
    Njd[1] = fmaf(rj.N[1], d[0], fmaf(rj.N[3], d[1], rj.N[4] * d[2]));
    Njd[2] = fmaf(rj.N[2], d[0], fmaf(rj.N[4], d[1], rj.N[5] * d[2]));
    const float ai = 0.5f * fmaf(d[0], Nid[0], fmaf(d[1], Nid[1], d[2] * Nid[2]));
    const float aj = 0.5f * fmaf(d[0], Njd[0], fmaf(d[1], Njd[1], d[2] * Njd[2]));
    const float bi = fmaf(ri.bb[0], d[0], fmaf(ri.bb[1], d[1], ri.bb[2] * d[2]));
    const float bj = fmaf(rj.bb[0], d[0], fmaf(rj.bb[1], d[1], rj.bb[2] * d[2]));
    const float dA = rj.A - ri.A;
    // x_bar: coefficient of d, then the N d and b_bar parts
    const float cd = K * (rj.V * fmaf(dA, bi, -ai) - ri.V * fmaf(-dA, bj, aj));
    const float gVj = G * rj.V, gVi = G * ri.V;
#pragma unroll
    for (int k = 0; k < DIM; ++k)
        xb[k] += cd * d[k] - gVj * Nid[k] - gVi * Njd[k] + dA * (gVj * ri.bb[k] + gVi * rj.bb[k]);
    vb = fmaf(G, fmaf(dA, bj, -aj), vb);
    ab = fmaf(-G, fmaf(ri.V, bj, rj.V * bi), ab);
}

