// wl_body.cuh -- device-side body description: signed-distance functions with analytic
// gradients, and the BDIM kernel moments (Eq. 1-2, "AutoBody ... signed-
// distance function as well as the coordinates mapping"; readings R-B, R-E).
// Independent restatement for the GPU path; shares nothing with oracle/.
#pragma once
#include "wl_common.cuh"

struct BodyP {
    int kind;        // WL_BODY_*
    int axis;        // torus / cylinder axis
    float R, r;      // sphere / cylinder radius R; torus major R / minor r
    float eps;       // BDIM kernel half-width
};

#define WLB_NONE 0
#define WLB_SPHERE 1
#define WLB_TORUS 2
#define WLB_CYLINDER 3

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

// Signed distance and unit normal at body-frame position xi (translation map: J = I).  T = double in measure!
// (a face 100 cells from the origin carries 6e-6 of fp32 round-off in its position, which mu0's slope 1/2eps turns
// into 3e-6 of mu0: evaluated in fp64 and rounded once, d is good to 6e-8), T = float elsewhere.
template <int ND, class T>
__device__ __forceinline__ T body_sdf(const BodyP& b, const T (&xi)[3], T (&nrm)[3])
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
