// wl_body.cuh -- device-side body description: signed-distance functions with analytic
// gradients, and the BDIM kernel moments (Eq. 1-2, "AutoBody ... signed-
// distance function as well as the coordinates mapping"; readings R-B, R-E).
// Independent restatement for the GPU path; shares nothing with oracle/.
#pragma once
#include "wl_common.cuh"

#define WLB_NONE 0
#define WLB_SPHERE 1
#define WLB_TORUS 2
#define WLB_CYLINDER 3
#define WLB_PLANE 4
#define WLB_MAXPART 4

// static description of one primitive of the body (the time-dependent part of its map lives in DevScal: PartState)
struct PartP {
    int kind;        // WL_BODY_*
    int axis;        // torus / cylinder / plane axis
    float R, r;      // sphere / cylinder radius R; torus major R / minor r
    float shell;     // > 0: thin shell |sdf| - shell
    float spin;      // angular velocity about the axis through the centre
    int scaled;      // the map has a non-rigid part (some scale_amp != 0): first-order distance d0 / |J^T grad sdf|
    int op;          // 0 union, 1 difference (with the body built from the primitives before it)
};
struct BodyP {
    int n;           // primitives (0: no body)
    PartP part[WLB_MAXPART];
    float eps;       // BDIM kernel half-width
    int general;     // the body velocity is a field (several primitives, a non-rigid map or spin): V array instead of three scalars
};

// cosine kernel K(s) = (1 + cos(pi s/eps)) / (2 eps) on |s| < eps
__device__ __forceinline__ float bdim_K(float s, float eps)
{
    if (fabsf(s) >= eps) return 0.0f;
    return (1.0f + cospif(s / eps)) / (2.0f * eps);
}
// zeroth moment mu0(d) = int_{-eps}^{d} K
__device__ __forceinline__ float bdim_mu0(float d, float eps)
{
    float a = d / eps;
    if (a <= -1.0f) return 0.0f;
    if (a >= 1.0f) return 1.0f;
    // near d = -eps the closed form cancels: with b = 1 + a, mu0 = (t - sin t)/(2 pi), t = pi b,
    // summed as a series so that tiny mu0 (which set the Poisson diagonal of nearly buried
    // cells) keep their relative accuracy in fp32
    float b = 1.0f + a;
    if (b < 0.16f) {
        float t = 3.14159265358979f * b, t2 = t * t;
        float ser = t * t2 * (1.0f / 6.0f - t2 * (1.0f / 120.0f - t2 * (1.0f / 5040.0f - t2 * (1.0f / 362880.0f))));
        return ser * 0.15915494309189535f;
    }
    return 0.5f + 0.5f * a + sinpif(a) * 0.15915494309189535f;
}
// first moment mu1(d) = int_{-d}^{eps} s K ds
__device__ __forceinline__ float bdim_mu1(float d, float eps)
{
    float a = d / eps;
    if (a <= -1.0f || a >= 1.0f) return 0.0f;
    float sp, cp;
    sincospif(a, &sp, &cp);
    return eps * (0.25f - 0.25f * a * a - (a * sp + (1.0f + cp) * 0.3183098861837907f) * 0.15915494309189535f);
}

// Signed distance and its gradient at body-frame position xi for one primitive.  T = double in measure! (a face 100 cells
// from the origin carries 6e-6 of fp32 round-off in its position, which mu0's slope 1/2eps turns into 3e-6 of mu0:
// evaluated in fp64 and rounded once, d is good to 6e-8), T = float elsewhere.
template <int ND, class T>
__device__ __forceinline__ T prim_sdf(const PartP& b, const T (&xi)[3], T (&nrm)[3])
{
    nrm[0] = nrm[1] = nrm[2] = T(0);
    const T tiny = T(1e-12);
    if (b.kind == WLB_SPHERE) {
        T rr = T(0);
#pragma unroll
        for (int k = 0; k < ND; ++k) rr += xi[k] * xi[k];
        rr = sqrt(rr);
        if (rr >= tiny) {
            T inv = T(1) / rr;
#pragma unroll
            for (int k = 0; k < ND; ++k) nrm[k] = xi[k] * inv;
        }
        return rr - (T)b.R;
    }
    if (b.kind == WLB_PLANE) {             // half-space below the plane through the centre, normal +e_axis
        nrm[b.axis] = T(1);
        return xi[b.axis];
    }
    // torus and cylinder: axis a, rho = distance from the axis
    T xa, xb, xc;
    if (b.axis == 0) { xa = xi[0]; xb = xi[1]; xc = xi[2]; }
    else if (b.axis == 1) { xa = xi[1]; xb = xi[2]; xc = xi[0]; }
    else { xa = xi[2]; xb = xi[0]; xc = xi[1]; }
    T rho = sqrt(xb * xb + xc * xc);
    if (b.kind == WLB_CYLINDER) {          // circular cylinder along the axis: d = rho - R, normal in the cross-plane
        T nb = T(0), nc = T(0);
        if (rho >= tiny) { T ir = T(1) / rho; nb = xb * ir; nc = xc * ir; }
        if (b.axis == 0) { nrm[1] = nb; nrm[2] = nc; }
        else if (b.axis == 1) { nrm[2] = nb; nrm[0] = nc; }
        else { nrm[0] = nb; nrm[1] = nc; }
        return rho - (T)b.R;
    }
    T w = rho - (T)b.R;
    T gq = sqrt(w * w + xa * xa);
    T na = T(0), nb = T(0), nc = T(0);
    if (gq >= tiny && rho >= tiny) {
        T ig = T(1) / gq, wr = (w * ig) / rho;
        na = xa * ig; nb = wr * xb; nc = wr * xc;
    } else if (gq >= tiny) {
        na = xa / gq;
    }
    if (b.axis == 0) { nrm[0] = na; nrm[1] = nb; nrm[2] = nc; }
    else if (b.axis == 1) { nrm[1] = na; nrm[2] = nb; nrm[0] = nc; }
    else { nrm[2] = na; nrm[0] = nb; nrm[1] = nc; }
    return gq - (T)b.r;
}

// The whole body at the point x (absolute grid coordinates), reading R-E3: for every primitive the map xi = s .* (x - c),
// the primitive's SDF (shell: |d0| - shell), normal J^T grad / |.| and first-order distance d0 / |J^T grad| when the map is
// non-rigid, velocity dc/dt - (ds/dt / s)(x - c) + spin e_a x (x - c); union = min, difference = max(d, -d_B), normal and
// velocity from the primitive that decides.  Returns d; fills nrm and vel.
template <int ND, class T>
__device__ __forceinline__ T body_eval(const BodyP& B, const PartState* __restrict__ st, const double (&x)[3], T (&nrm)[3], float (&vel)[3])
{
    T d = T(1e30);
    nrm[0] = nrm[1] = nrm[2] = T(0);
    vel[0] = vel[1] = vel[2] = 0.0f;
    for (int e = 0; e < B.n; ++e) {
        const PartP& p = B.part[e];
        const PartState& q = st[e];
        T xi[3] = { T(0), T(0), T(0) }, g[3];
        double rel[3] = { 0.0, 0.0, 0.0 };
#pragma unroll
        for (int k = 0; k < ND; ++k) { rel[k] = x[k] - q.c[k]; xi[k] = (T)(q.s[k] * rel[k]); }
        T d0 = prim_sdf<ND, T>(p, xi, g);
        if (p.shell > 0.0f) {
            const T sg = d0 < T(0) ? T(-1) : T(1);
            d0 = fabs(d0) - (T)p.shell;
#pragma unroll
            for (int k = 0; k < 3; ++k) g[k] *= sg;
        }
        if (p.scaled) {
            T m = T(0);
#pragma unroll
            for (int k = 0; k < ND; ++k) { g[k] *= (T)q.s[k]; m += g[k] * g[k]; }
            m = sqrt(m);
            if (m >= T(1e-12)) {
                const T im = T(1) / m;
                d0 *= im;
#pragma unroll
                for (int k = 0; k < ND; ++k) g[k] *= im;
            } else {
                g[0] = g[1] = g[2] = T(0);
            }
        }
        if (p.op == 1) {
            d0 = -d0;
#pragma unroll
            for (int k = 0; k < 3; ++k) g[k] = -g[k];
        }
        const bool take = e == 0 || (p.op == 1 ? d0 > d : d0 < d);
        if (take) {
            d = d0;
#pragma unroll
            for (int k = 0; k < 3; ++k) nrm[k] = g[k];
            float v[3] = { 0.f, 0.f, 0.f };
#pragma unroll
            for (int k = 0; k < ND; ++k) v[k] = (float)((double)q.cdot[k] - (double)q.sdot_s[k] * rel[k]);
            if (p.spin != 0.0f) {
                const int a = ND == 3 ? p.axis : 2, b1 = (a + 1) % 3, c1 = (a + 2) % 3;
                if (b1 < ND) v[b1] += (float)(-(double)p.spin * rel[c1]);
                if (c1 < ND) v[c1] += (float)((double)p.spin * rel[b1]);
            }
#pragma unroll
            for (int k = 0; k < 3; ++k) vel[k] = v[k];
        }
    }
    return d;
}
