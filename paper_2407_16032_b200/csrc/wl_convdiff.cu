// wl_convdiff.cu -- conv_diff! fused with the BDIM blend and the Heun average (scale_u!).
//   r_i = -d_j(u_j u_i) + nu d_jj u_i      conservative fluxes, flux-limited QUICK + central
//                                          diffusion (Eq. 1; R-G, R-H, R-I)
//   f   = u0 + dt r - V ;  B_i = V_i + mu0 f_i + sum_j mu1_ij (f_i[c+d_j] - f_i[c-d_j])/2
//                                          (Eq. 1-2; R-B, R-C)
//   predictor: u = B ; corrector: u = (u' + B)/2            (P:76, P:139 scale_u!; R-K, R-L)
// One pass over the grid: f is never stored.  mu1 is non-zero only within eps of the body
// surface; only there the neighbours' f (six more evaluations of r) are recomputed.
#include <cstdio>
#include "wl_internal.h"

__device__ __forceinline__ float med3(float a, float b, float c)
{
    return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c));
}
// limited third-order upwind face value q(U,C,D) (R-G)
__device__ __forceinline__ float quick(float U, float C, float D)
{
    return med3((5.0f * C + 2.0f * D - U) * (1.0f / 6.0f), C, med3(10.0f * C - 9.0f * U, C, D));
}

// Per-thread stencil addressing: lin[d][k] = stride_d * wrap_d(c_d + k - 2), k = 0..4.
template <int ND>
struct Sten {
    int64_t lin[3][5];
    int c[3];
    __device__ __forceinline__ void set(const Grid& g, int c0, int c1, int c2)
    {
        c[0] = c0; c[1] = c1; c[2] = c2;
        const int64_t st[3] = { 1, g.sy, g.sz };
#pragma unroll
        for (int d = 0; d < 3; ++d)
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                int cc = d < ND ? wrapc(c[d] + k - 2, g.n[d], g.per[d]) : 0;
                // non-periodic: clamp into the padded array; clamped entries are never used
                if (d < ND) { if (cc < 0) cc = 0; if (cc > g.n[d] + 1) cc = g.n[d] + 1; }
                lin[d][k] = (int64_t)cc * st[d];
            }
    }
    // offset of c + a e_0 + b e_1 + cc e_2 (|.| <= 2)
    __device__ __forceinline__ int64_t at(int a, int b, int cc) const
    {
        return (int64_t)WL_OFF + lin[0][a + 2] + lin[1][b + 2] + lin[2][cc + 2];
    }
};

// Flux through the lower j-boundary of the control volume of w_i at c + s e_j (s = 0 or 1):
//   phi = (w_j[c-d_i] + w_j[c])/2 ; PHI = phi psi - nu (w_i[c] - w_i[c-d_j])
template <int ND, int I, int J>
__device__ __forceinline__ float flux(const FlowP& P, const float* __restrict__ w, const Sten<ND>& S, int s)
{
    const Grid& g = P.g;
    const float* wi = w + I * g.nalloc;
    const float* wj = w + J * g.nalloc;
    int o[3] = { 0, 0, 0 };
    o[J] = s;
    int om[3] = { o[0], o[1], o[2] };       // c - d_j
    om[J] -= 1;
    int oi[3] = { o[0], o[1], o[2] };       // c - d_i
    oi[I] -= 1;
    float phi = 0.5f * (wj[S.at(oi[0], oi[1], oi[2])] + wj[S.at(o[0], o[1], o[2])]);
    float wc = wi[S.at(o[0], o[1], o[2])];
    float wm = wi[S.at(om[0], om[1], om[2])];
    const bool pos = phi > 0.0f;
    const int cj = S.c[J] + s;
    const int N = g.n[J];
    const bool fb = !g.per[J] && (pos ? (cj <= 1 + (I == J ? 1 : 0)) : (cj >= N + 1));
    int ou[3] = { o[0], o[1], o[2] };
    ou[J] += fb ? 0 : (pos ? -2 : 1);
    // the far-upwind value: c - 2 d_j (phi > 0) or c + d_j; the offset stays within +-2 of c
    float wu;
    {
        // ou[J] is in {s-2, s, s+1} subset of [-2, 2]
        int64_t a = (int64_t)WL_OFF;
#pragma unroll
        for (int d = 0; d < 3; ++d) a += S.lin[d][ou[d] + 2];
        wu = wi[a];
    }
    float C = pos ? wm : wc, D = pos ? wc : wm;
    float psi = fb ? 0.5f * (wm + wc) : quick(wu, C, D);
    return phi * psi - P.nu * (wc - wm);
}

template <int ND, int I>
__device__ __forceinline__ float rhs_comp(const FlowP& P, const float* __restrict__ w, const Sten<ND>& S)
{
    float acc = flux<ND, I, 0>(P, w, S, 0) - flux<ND, I, 0>(P, w, S, 1);
    acc += flux<ND, I, 1>(P, w, S, 0) - flux<ND, I, 1>(P, w, S, 1);
    if (ND == 3) acc += flux<ND, I, 2>(P, w, S, 0) - flux<ND, I, 2>(P, w, S, 1);
    return acc;
}

// f_i at an arbitrary padded position (used only inside the mu1 band):
// ghost in a non-periodic direction -> r = 0; otherwise r at the wrapped position.
template <int ND, int I>
__device__ float f_at(const FlowP& P, const float* __restrict__ w, const float* __restrict__ u0, float dt, float Vi,
                      int c0, int c1, int c2)
{
    const Grid& g = P.g;
    int c[3] = { c0, c1, c2 };
    bool ghost = false;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        if (g.per[d]) c[d] = wrapc(c[d], g.n[d], 1);
        else if (c[d] < 1 || c[d] > g.n[d]) ghost = true;
    }
    float r = 0.0f;
    if (!ghost) {
        Sten<ND> S;
        S.set(g, c[0], c[1], c[2]);
        r = rhs_comp<ND, I>(P, w, S);
    }
    return u0[I * g.nalloc + gidx(g, c[0], c[1], c[2])] + dt * r - Vi;
}

template <int ND, int I>
__device__ __forceinline__ void blend_comp(const FlowP& P, const float* __restrict__ w, const float* __restrict__ u0,
                                           const float* __restrict__ mu0, const float* __restrict__ mu1,
                                           float* __restrict__ out, const Sten<ND>& S, int64_t id, float dt, float Vi, int corrector)
{
    const Grid& g = P.g;
    float r = rhs_comp<ND, I>(P, w, S);
    float f = u0[I * g.nalloc + id] + dt * r - Vi;
    float B = Vi + mu0[I * g.nalloc + id] * f;
    float m1[3];
    bool band = false;
#pragma unroll
    for (int j = 0; j < ND; ++j) {
        m1[j] = mu1[(I * ND + j) * g.nalloc + id];
        band = band || (m1[j] != 0.0f);
    }
    if (band) {
#pragma unroll
        for (int j = 0; j < ND; ++j) {
            int cp[3] = { S.c[0], S.c[1], S.c[2] }, cm[3] = { S.c[0], S.c[1], S.c[2] };
            cp[j] += 1; cm[j] -= 1;
            float fp = f_at<ND, I>(P, w, u0, dt, Vi, cp[0], cp[1], cp[2]);
            float fm = f_at<ND, I>(P, w, u0, dt, Vi, cm[0], cm[1], cm[2]);
            B += m1[j] * 0.5f * (fp - fm);
        }
    }
    out[I * g.nalloc + id] = corrector ? 0.5f * (w[I * g.nalloc + id] + B) : B;
}

template <int ND>
__global__ void __launch_bounds__(512) k_conv_diff_bdim(FlowP P, Tiling T, const float* __restrict__ w, const float* __restrict__ u0,
                                                        const float* __restrict__ mu0, const float* __restrict__ mu1,
                                                        float* __restrict__ out, const DevScal* __restrict__ ds, int corrector)
{
    const Grid& g = P.g;
    const float dt = ds->dt;
    const float V0 = ds->vel[0], V1 = ds->vel[1], V2 = ds->vel[2];
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        Sten<ND> S;
        S.set(g, c0, c1, c2);
        blend_comp<ND, 0>(P, w, u0, mu0, mu1, out, S, id, dt, V0, corrector);
        blend_comp<ND, 1>(P, w, u0, mu0, mu1, out, S, id, dt, V1, corrector);
        if (ND == 3) blend_comp<ND, 2>(P, w, u0, mu0, mu1, out, S, id, dt, V2, corrector);
        // the corrector leaves the convective-exit plane at the predictor's value (R-N); the
        // output is another buffer, so carry the plane over
        if (corrector && P.exit_bc && c0 == g.n[0]) out[id + 1] = w[id + 1];
    }
}

void wl_k_conv_diff_bdim(wl_sim* s, const float* w, const float* u0, float* out, int corrector)
{
    FlowP P = wl_flowp(s);
    Tiling T = wl_tiles_interior(s, P.g);
    ProfScope ps(s, WLK_CONVDIFF);
    if (s->nd == 3)
        k_conv_diff_bdim<3><<<wl_grid(s, T), wl_block(3), 0, s->st>>>(P, T, w, u0, s->mu0, s->mu1, out, s->ds, corrector);
    else
        k_conv_diff_bdim<2><<<wl_grid(s, T), wl_block(2), 0, s->st>>>(P, T, w, u0, s->mu0, s->mu1, out, s->ds, corrector);
}
