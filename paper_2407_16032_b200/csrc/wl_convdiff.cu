// wl_convdiff.cu -- conv_diff! fused with the BDIM blend and the Heun average (scale_u!).
//   r_i = -d_j(u_j u_i) + nu d_jj u_i      conservative fluxes, flux-limited QUICK + central
//                                          diffusion (Eq. 1; R-G, R-H, R-I)
//   f   = u0 + dt r - V ;  B_i = V_i + mu0 f_i + sum_j mu1_ij (f_i[c+d_j] - f_i[c-d_j])/2
//                                          (Eq. 1-2; R-B, R-C)
//   predictor: u = B ; corrector: u = (u' + B)/2            (P:76, P:139 scale_u!; R-K, R-L)
// f is never stored.  Kernels:
//  * k_cd_tile3 (3-D, x and y not periodic: every inflow/outflow case) and k_cd_tile2 (everything else): the whole grid.
//    A block of 256 x ND threads owns a 128 x 8 column of cells and marches along z; the velocity components of the five
//    planes z-2..z+2 (two-cell halo in x and y) sit in a shared-memory ring, so every value is read from HBM/L2 once per
//    tile and all stencil reads are conflict-free 16-byte shared loads.  A thread owns four consecutive x cells of ONE
//    component; every limited face flux is computed once (x faces inside the thread, y faces handed down through shared
//    memory, z faces kept for the next plane).  k_cd_tile3 fills the ring with TMA boxes, k_cd_tile2 through registers
//    with the periodic wrap applied while loading.  They write u = V + mu0 f (with the Heun average in the corrector)
//    and never read mu1.
//  * k_cd_band: mu1 is non-zero only within eps of the body surface; measure! leaves a compact list of those faces
//    (wl_flow.cu) and this kernel adds sum_j mu1_ij (f_i[c+d_j]-f_i[c-d_j])/2 there, recomputing the six neighbouring
//    r from global memory (flux / rhs_comp / f_at below).
#include <cstdio>
#include <cstdlib>
#include "wl_internal.h"
#include "wl_tma.cuh"

__device__ __forceinline__ float med3(float a, float b, float c)
{
    return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c));
}
// limited third-order upwind face value q(U,C,D) = median((5C+2D-U)/6, C, median(10C-9U, C, D)) (R-G), written in
// differences from C: with d = D-C, x = 9(C-U), y = (2d + (C-U))/6 and s = sign(d),
//     q = C + s max(0, min(s y, s x, |d|))
// (the inner median clamps x to [0,d], the outer one clamps y to [0, inner]; for d < 0 everything mirrors).  Three
// min/max on the half-rate ALU pipe instead of eight; the products with s = +-1 are exact.
__device__ __forceinline__ float quick(float U, float C, float D)
{
    const float d = D - C, t = C - U;
    const float x = 9.0f * t, y = (2.0f * d + t) * (1.0f / 6.0f);
    const float s = copysignf(1.0f, d);
    const float m = fmaxf(0.0f, fminf(fminf(s * y, s * x), fabsf(d)));
    return fmaf(s, m, C);
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
    const int64_t id = gidx(g, c[0], c[1], c[2]);
    if (P.Vf) Vi = P.Vf[I * g.nalloc + id];          // a general body: V at THIS face
    return u0[I * g.nalloc + id] + dt * r - Vi;
}


// ====================================================================== the tile kernel
#define CD_TX 32                       // threads along x, four cells each
#define CD2_TY 8                       // rows per block of k_cd_tile2 (one block of 256 x ND threads per SM)
#define CD3_TY 4                       // rows per block of k_cd_tile3: two resident blocks of 128 x 3 threads beat one of 256 x 3 (630 -> 587 us on C4)
#define CD_TY CD2_TY                   // the register-staged loaders below belong to k_cd_tile2
#define CD_NT (CD_TX * CD_TY)
#define CD_G (CD_TX + 2)               // float4 groups per shared row: cells bx-4 .. bx+4*CD_TX+3
#define CD_W (4 * CD_G)                // floats per shared row
#define CD_R (CD_TY + 4)               // shared rows: by-2 .. by+CD_TY+1
#define CD_PLANE (CD_W * CD_R)         // floats per component per plane
#define CD3_NT (CD_TX * CD3_TY)        // the same for k_cd_tile3
#define CD3_R (CD3_TY + 4)
#define CD3_PLANE (CD_W * CD3_R)
#define CD_NP 5                        // ring of planes z-2 .. z+2

__device__ __forceinline__ int wrap_any(int c, int N)      // 1..N for any c
{
    int m = (c - 1) % N;
    return (m < 0 ? m + N : m) + 1;
}
__device__ __forceinline__ int src_coord(int c, int N, int per)
{
    if (per) return wrap_any(c, N);
    return c < 0 ? 0 : (c > N + 1 ? N + 1 : c);   // clamped values are never used (R-H fallback)
}

// One 16-byte group of a shared plane: component comp, shared row `row`, group grp, plane cz.
template <int ND>
__device__ __forceinline__ float4 cd_fetch(const Grid& g, const float* __restrict__ w, int item, int bx, int by, int cz)
{
    const int comp = item / (CD_R * CD_G);
    const int rem = item - comp * (CD_R * CD_G);
    const int row = rem / CD_G, grp = rem - row * CD_G;
    const int cy = src_coord(by - 2 + row, g.n[1], g.per[1]);
    const int xs = bx - 4 + 4 * grp;
    const float* src = w + comp * g.nalloc + (int64_t)WL_OFF + (int64_t)cy * g.sy + (int64_t)cz * g.sz;
    if (xs >= 1 && xs + 3 <= g.n[0]) return ld4(src, xs);
    float4 v;
    v.x = __ldg(src + src_coord(xs, g.n[0], g.per[0]));
    v.y = __ldg(src + src_coord(xs + 1, g.n[0], g.per[0]));
    v.z = __ldg(src + src_coord(xs + 2, g.n[0], g.per[0]));
    v.w = __ldg(src + src_coord(xs + 3, g.n[0], g.per[0]));
    return v;
}

#define CD_ITEMS(ND) ((ND) * CD_R * CD_G)
// limited flux through one face: wm | wc are the values either side, wup / wun the far-upwind
// values for phi > 0 / phi <= 0, fbp / fbn the boundary fallbacks of R-H
__device__ __forceinline__ float face_flux(float phi, float wup, float wm, float wc, float wun, bool fbp, bool fbn, float nu)
{
    // phi psi - nu (wc - wm) with the limited value psi = q(U, C, D) of the upwind triple, written WITHOUT selecting U, C, D: with
    // d1 = wc - wm, tt = the difference on the upwind side (wm - wup if phi > 0, else wun - wc), s1 = sign(d1) and avg = (wm + wc)/2,
    //     m = max(0, min((2 |d1| + s1 tt)/6, 9 s1 tt, |d1|)),   psi = avg +- (s1 m - d1/2)   (+ for phi > 0),
    // (the quick() above in differences from C, and C = avg -+ d1/2), so phi psi = phi avg + |phi| (s1 m - d1/2): one select, two sign
    // transfers, and the three differences of a row of faces are shared between neighbouring faces.  The R-H fallback drops the
    // correction.
    const bool pos = phi > 0.0f;
    const bool fb = pos ? fbp : fbn;
    const float d1 = wc - wm;
    const float tt = pos ? wm - wup : wun - wc;
    const unsigned sgn = __float_as_uint(d1) & 0x80000000u;
    const float stt = __uint_as_float(__float_as_uint(tt) ^ sgn);
    const float ad = fabsf(d1);
    const float m = fmaxf(0.0f, fminf(fminf(fmaf(stt, 1.0f / 6.0f, ad * (1.0f / 3.0f)), 9.0f * stt), ad));
    float corr = fmaf(-0.5f, d1, __uint_as_float(__float_as_uint(m) ^ sgn));
    corr = fb ? 0.0f : corr;
    return fmaf(0.5f * phi, wm + wc, fmaf(fabsf(phi), corr, -nu * d1));
}

struct CdT { int ntx, nty, ntz, ntiles, zc; };

// ====================================================================== the tile kernel, one component per thread
// (a) a thread owns four cells of ONE component (blocks of 256 x ND threads; warps are component-uniform), (b) the flux
// through a y face is computed once, by the thread above it, and handed down through shared memory, (c) the flux through
// the upper z face is kept for the next plane of the march, where it is the lower one.  41 instead of 63 fluxes per four
// cells of the three components (a flux is the same expression of the same operands whichever thread evaluates it).
// view of the ring for one thread: b[dz + 2] points at the thread's own float4 of component 0 in plane z+dz, so that
// every stencil read is one shared load at a compile-time offset (component, row and group offsets are immediates)
// (TY: rows per block, which fixes the distance between the components of a plane)
template <int TY>
struct CdView2 { const float* b[CD_NP]; };
template <int TY>
__device__ __forceinline__ void v4(const CdView2<TY>& v, int comp, int dz, int dy, int dg, float* o)
{
    const float4 t = *reinterpret_cast<const float4*>(v.b[dz + 2] + comp * (CD_W * (TY + 4)) + dy * CD_W + 4 * dg);
    o[0] = t.x; o[1] = t.y; o[2] = t.z; o[3] = t.w;
}
template <int TY>
__device__ __forceinline__ float v1(const CdView2<TY>& v, int comp, int dz, int dy, int col)
{
    return v.b[dz + 2][comp * (CD_W * (TY + 4)) + dy * CD_W + col];
}
#define CD2_NT(ND) (CD_NT * (ND))
#define CD2_STAGE(ND) ((CD_ITEMS(ND) + CD2_NT(ND) - 1) / CD2_NT(ND))

template <int ND>
__device__ __forceinline__ void cd2_load_regs(const Grid& g, const float* __restrict__ w, int bx, int by, int cz, float4 (&st)[CD2_STAGE(ND)])
{
#pragma unroll
    for (int k = 0; k < CD2_STAGE(ND); ++k) {
        const int item = threadIdx.x + k * CD2_NT(ND);
        if (item < CD_ITEMS(ND)) st[k] = cd_fetch<ND>(g, w, item, bx, by, cz);
    }
}
template <int ND>
__device__ __forceinline__ void cd2_store_regs(float* __restrict__ slot, const float4 (&st)[CD2_STAGE(ND)])
{
#pragma unroll
    for (int k = 0; k < CD2_STAGE(ND); ++k) {
        const int item = threadIdx.x + k * CD2_NT(ND);
        if (item < CD_ITEMS(ND)) reinterpret_cast<float4*>(slot)[item] = st[k];
    }
}

// what a thread carries from the flux phase to the output phase of a plane
struct Cd2Part {
    float rx[4];     // F_x[k] - F_x[k+1]
    float fyl[4];    // flux through the lower y face (handed to the thread below as its upper one)
    float fyu[4];    // flux through the upper y face: computed here only in the top row of the block
    float fzd[4];    // F_z lower - F_z upper
    float wc[5];     // w_I at the own cells and the next one (convective-exit carry)
};

// fluxes of component I at the thread's four cells of plane gz.  fz: in (unless `first`) the flux through the lower z
// face left by the previous plane; out the flux through the upper z face.
template <int ND, int I, int TY>
__device__ __forceinline__ void cd2_fluxes(const FlowP& P, const CdView2<TY>& v, int gx, int gy, int gz, bool top, bool first, float (&fz)[4], Cd2Part& o)
{
    const Grid& g = P.g;
    const float nu = P.nu;
    float a[12];
    v4(v, I, 0, 0, -1, a); v4(v, I, 0, 0, 0, a + 4); v4(v, I, 0, 0, 1, a + 8);
#pragma unroll
    for (int k = 0; k < 5; ++k) o.wc[k] = a[4 + k];
    // ---- x faces gx .. gx+4 (shared between the thread's cells)
    {
        float px[5];
        if (I == 0) {
#pragma unroll
            for (int f = 0; f < 5; ++f) px[f] = 0.5f * (a[3 + f] + a[4 + f]);
        } else {
            float lo[5], hi[5];
            v4(v, 0, 0, 0, 0, hi); hi[4] = v1(v, 0, 0, 0, 4);
            if (I == 1) { v4(v, 0, 0, -1, 0, lo); lo[4] = v1(v, 0, 0, -1, 4); }
            else        { v4(v, 0, -1, 0, 0, lo); lo[4] = v1(v, 0, -1, 0, 4); }
#pragma unroll
            for (int f = 0; f < 5; ++f) px[f] = 0.5f * (lo[f] + hi[f]);
        }
        float F[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            const int cj = gx + f;
            const bool fbp = !g.per[0] && cj <= 1 + (I == 0 ? 1 : 0), fbn = !g.per[0] && cj >= g.n[0] + 1;
            F[f] = face_flux(px[f], a[2 + f], a[3 + f], a[4 + f], a[5 + f], fbp, fbn, nu);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) o.rx[k] = F[k] - F[k + 1];
    }
    // ---- y faces: the lower one (gy) always, the upper one (gy+1) in the top row of the block only
    {
        float m2[4], m1[4], p1[4], pl[4];
        v4(v, I, 0, -2, 0, m2); v4(v, I, 0, -1, 0, m1); v4(v, I, 0, 1, 0, p1);
        float b0[4], c0[4], e0 = 0.0f;
        if (I == 1) {
#pragma unroll
            for (int k = 0; k < 4; ++k) pl[k] = 0.5f * (m1[k] + a[4 + k]);
        } else if (I == 0) {
            v4(v, 1, 0, 0, 0, b0); e0 = v1(v, 1, 0, 0, -1);
#pragma unroll
            for (int k = 0; k < 4; ++k) pl[k] = 0.5f * ((k == 0 ? e0 : b0[k == 0 ? 0 : k - 1]) + b0[k]);
        } else {
            v4(v, 1, -1, 0, 0, b0); v4(v, 1, 0, 0, 0, c0);
#pragma unroll
            for (int k = 0; k < 4; ++k) pl[k] = 0.5f * (b0[k] + c0[k]);
        }
        const bool np = !g.per[1];
        const bool lfbp = np && gy <= 1 + (I == 1 ? 1 : 0), lfbn = np && gy >= g.n[1] + 1;
#pragma unroll
        for (int k = 0; k < 4; ++k) o.fyl[k] = face_flux(pl[k], m2[k], m1[k], a[4 + k], p1[k], lfbp, lfbn, nu);
        if (top) {
            float p2[4], pu[4], b1[4], c1[4];
            v4(v, I, 0, 2, 0, p2);
            if (I == 1) {
#pragma unroll
                for (int k = 0; k < 4; ++k) pu[k] = 0.5f * (a[4 + k] + p1[k]);
            } else if (I == 0) {
                v4(v, 1, 0, 1, 0, b1);
                const float e1 = v1(v, 1, 0, 1, -1);
#pragma unroll
                for (int k = 0; k < 4; ++k) pu[k] = 0.5f * ((k == 0 ? e1 : b1[k == 0 ? 0 : k - 1]) + b1[k]);
            } else {
                v4(v, 1, -1, 1, 0, b1); v4(v, 1, 0, 1, 0, c1);
#pragma unroll
                for (int k = 0; k < 4; ++k) pu[k] = 0.5f * (b1[k] + c1[k]);
            }
            const bool ufbp = np && gy + 1 <= 1 + (I == 1 ? 1 : 0), ufbn = np && gy + 1 >= g.n[1] + 1;
#pragma unroll
            for (int k = 0; k < 4; ++k) o.fyu[k] = face_flux(pu[k], m1[k], a[4 + k], p1[k], p2[k], ufbp, ufbn, nu);
        }
    }

    // ---- z faces: the upper one (gz+1) always; the lower one (gz) only on the first plane of the march
    if (ND == 3) {
        float m1[4], p1[4], p2[4], pu[4];
        v4(v, I, -1, 0, 0, m1); v4(v, I, 1, 0, 0, p1); v4(v, I, 2, 0, 0, p2);
        const bool np = !g.per[2];
        if (first) {
            float m2[4], pl[4], b0[4], c0[4];
            v4(v, I, -2, 0, 0, m2);
            if (I == 2) {
#pragma unroll
                for (int k = 0; k < 4; ++k) pl[k] = 0.5f * (m1[k] + a[4 + k]);
            } else if (I == 0) {
                v4(v, 2, 0, 0, 0, b0);
                const float e0 = v1(v, 2, 0, 0, -1);
#pragma unroll
                for (int k = 0; k < 4; ++k) pl[k] = 0.5f * ((k == 0 ? e0 : b0[k == 0 ? 0 : k - 1]) + b0[k]);
            } else {
                v4(v, 2, 0, -1, 0, b0); v4(v, 2, 0, 0, 0, c0);
#pragma unroll
                for (int k = 0; k < 4; ++k) pl[k] = 0.5f * (b0[k] + c0[k]);
            }
            const bool lfbp = np && gz <= 1 + (I == 2 ? 1 : 0), lfbn = np && gz >= g.n[2] + 1;
#pragma unroll
            for (int k = 0; k < 4; ++k) fz[k] = face_flux(pl[k], m2[k], m1[k], a[4 + k], p1[k], lfbp, lfbn, nu);
        }
        float b1[4], c1[4];
        if (I == 2) {
#pragma unroll
            for (int k = 0; k < 4; ++k) pu[k] = 0.5f * (a[4 + k] + p1[k]);
        } else if (I == 0) {
            v4(v, 2, 1, 0, 0, b1);
            const float e1 = v1(v, 2, 1, 0, -1);
#pragma unroll
            for (int k = 0; k < 4; ++k) pu[k] = 0.5f * ((k == 0 ? e1 : b1[k == 0 ? 0 : k - 1]) + b1[k]);
        } else {
            v4(v, 2, 1, -1, 0, b1); v4(v, 2, 1, 0, 0, c1);
#pragma unroll
            for (int k = 0; k < 4; ++k) pu[k] = 0.5f * (b1[k] + c1[k]);
        }
        const bool ufbp = np && gz + 1 <= 1 + (I == 2 ? 1 : 0), ufbn = np && gz + 1 >= g.n[2] + 1;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float up = face_flux(pu[k], m1[k], a[4 + k], p1[k], p2[k], ufbp, ufbn, nu);
            o.fzd[k] = fz[k] - up;
            fz[k] = up;
        }
    }
}

// what the output phase needs from global memory: issued BEFORE the flux phase of the plane, so that the L2 latency of these
// loads (they were the largest stall of the kernel: 1.8 warps per issue on the long scoreboard) hides behind the arithmetic
struct Cd2Pre { float mm[4], uu[4], vv[4]; };
template <int ND, int I>
__device__ __forceinline__ void cd2_preload(const FlowP& P, int gx, int gy, int gz, int nv, const float* __restrict__ u0,
                                            const float* __restrict__ mu0, float Vi, int corrector, Cd2Pre& o)
{
    const Grid& g = P.g;
#pragma unroll
    for (int k = 0; k < 4; ++k) { o.mm[k] = 0.0f; o.uu[k] = 0.0f; o.vv[k] = Vi; }
    if (nv <= 0) return;
    const int64_t id = gidx(g, gx, gy, gz);
    unpack4(ld4(mu0 + I * g.nalloc, id), o.mm);
    if (corrector) unpack4(ld4(u0 + I * g.nalloc, id), o.uu);
    if (P.Vf) unpack4(ld4(P.Vf + I * g.nalloc, id), o.vv);      // a general body: V is a field
}

// output phase: r = rx + (fyl - fyu) + fzd; f = u0 + dt r - V; B = V + mu0 f; predictor u = B, corrector u = (u' + B)/2
template <int ND, int I>
__device__ __forceinline__ void cd2_output(const FlowP& P, int gx, int gy, int gz, int nv, const Cd2Part& q, const float (&fyu)[4],
                                           const Cd2Pre& pre, float* __restrict__ out, float dt, int corrector)
{
    const Grid& g = P.g;
    if (nv <= 0) return;
    float o[4];
    const int64_t id = gidx(g, gx, gy, gz);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float r = q.rx[k];
        r += q.fyl[k] - fyu[k];
        if (ND == 3) r += q.fzd[k];
        const float uu = corrector ? pre.uu[k] : q.wc[k];
        const float f = uu + dt * r - pre.vv[k];
        const float B = pre.vv[k] + pre.mm[k] * f;
        o[k] = corrector ? 0.5f * (q.wc[k] + B) : B;
    }
    st4(out + I * g.nalloc, id, o, nv);
    if (I == 0 && corrector && P.exit_bc) {       // the corrector carries the convective-exit plane over (R-N)
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (gx + k == g.n[0]) out[id + k + 1] = q.wc[k + 1];
    }
}

template <int ND>
__global__ void __launch_bounds__(CD2_NT(ND), 1) k_cd_tile2(FlowP P, CdT T, const float* __restrict__ w, const float* __restrict__ u0,
                                                            const float* __restrict__ mu0, float* __restrict__ out,
                                                            const DevScal* __restrict__ ds, int corrector)
{
    extern __shared__ float4 cd_smem[];
    float* ring = reinterpret_cast<float*>(cd_smem);
    const Grid& g = P.g;
    const float dt = ds->dt;
    constexpr int NP = ND == 3 ? CD_NP : 1;
    constexpr int SLOT = ND * CD_PLANE;            // floats per ring slot
    float4* ex = reinterpret_cast<float4*>(ring + NP * SLOT);      // [ND][CD_TY][CD_TX] lower-y-face fluxes of the plane
    const int comp = threadIdx.x / CD_NT, t2 = threadIdx.x - comp * CD_NT;
    const float Vi = ds->vel[comp];
    CdView2<CD2_TY> v;
    const int tx = t2 & (CD_TX - 1), ty = t2 / CD_TX;
    const int tofs = (ty + 2) * CD_W + 4 * (tx + 1);          // the thread's own group inside a plane
    const bool top = ty == CD_TY - 1;
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        const int tix = tile % T.ntx, rem = tile / T.ntx;
        const int tiy = rem % T.nty, tiz = rem / T.nty;
        const int bx = 1 + 4 * CD_TX * tix, by = 1 + CD_TY * tiy;
        const int z0 = ND == 3 ? 1 + T.zc * tiz : 0;
        const int z1 = ND == 3 ? min(z0 + T.zc - 1, g.n[2]) : 0;
        const int gx = bx + 4 * tx, gy = by + ty;
        int nv = g.n[0] - gx + 1;
        nv = nv > 4 ? 4 : nv;
        if (gy > g.n[1]) nv = 0;
        __syncthreads();                           // the previous tile's reads are done
        {
            float4 st[CD2_STAGE(ND)];
#pragma unroll 1
            for (int d = 0; d < NP; ++d) {
                const int cz = ND == 3 ? src_coord(z0 - 2 + d, g.n[2], g.per[2]) : 0;
                cd2_load_regs<ND>(g, w, bx, by, cz, st);
                cd2_store_regs<ND>(ring + d * SLOT, st);
            }
        }
        __syncthreads();
        int s0 = 0;                                // ring slot of plane z-2
        float fz[4] = { 0.f, 0.f, 0.f, 0.f };      // flux through the upper z face of the previous plane
#pragma unroll 1
        for (int z = z0; z <= z1; ++z) {
            float4 st[CD2_STAGE(ND)];
            const bool more = ND == 3 && z < z1;
            if (more) cd2_load_regs<ND>(g, w, bx, by, src_coord(z + 3, g.n[2], g.per[2]), st);
#pragma unroll
            for (int d = 0; d < NP; ++d) {
                int s = s0 + d;
                if (s >= NP) s -= NP;
                v.b[ND == 3 ? d : 2] = ring + s * SLOT + tofs;
            }
            Cd2Part q;
            Cd2Pre pre;
            const bool first = z == z0;
            if (comp == 0)      { cd2_preload<ND, 0>(P, gx, gy, z, nv, u0, mu0, Vi, corrector, pre); cd2_fluxes<ND, 0>(P, v, gx, gy, z, top, first, fz, q); }
            else if (comp == 1) { cd2_preload<ND, 1>(P, gx, gy, z, nv, u0, mu0, Vi, corrector, pre); cd2_fluxes<ND, 1>(P, v, gx, gy, z, top, first, fz, q); }
            else if (ND == 3)   { cd2_preload<ND, 2>(P, gx, gy, z, nv, u0, mu0, Vi, corrector, pre); cd2_fluxes<ND, 2>(P, v, gx, gy, z, top, first, fz, q); }
            ex[(comp * CD_TY + ty) * CD_TX + tx] = make_float4(q.fyl[0], q.fyl[1], q.fyl[2], q.fyl[3]);
            __syncthreads();                       // every lower-y-face flux of the plane is in shared memory
            float fyu[4];
            if (top) {
#pragma unroll
                for (int k = 0; k < 4; ++k) fyu[k] = q.fyu[k];
            } else {
                unpack4(ex[(comp * CD_TY + ty + 1) * CD_TX + tx], fyu);
            }
            if (comp == 0)      cd2_output<ND, 0>(P, gx, gy, z, nv, q, fyu, pre, out, dt, corrector);
            else if (comp == 1) cd2_output<ND, 1>(P, gx, gy, z, nv, q, fyu, pre, out, dt, corrector);
            else if (ND == 3)   cd2_output<ND, 2>(P, gx, gy, z, nv, q, fyu, pre, out, dt, corrector);
            if (more) {
                __syncthreads();
                cd2_store_regs<ND>(ring + s0 * SLOT, st);
                s0 = s0 + 1 == NP ? 0 : s0 + 1;
                __syncthreads();
            }
        }
    }
}

// ---- k_cd_tile3: k_cd_tile2 with the ring filled by the TMA engine (3-D, non-periodic x and y).
// A ring of SIX plane slots: while plane z is computed from the planes z-2 .. z+2, the box copies of plane z+3 (one
// per component: cells bx-4 .. bx+131 of rows by-2 .. by+9, out-of-range parts zero-filled; z wraps through the plane
// coordinate) land in the sixth slot, issued by one thread a whole plane ahead and completing on the slot's mbarrier.
// No thread touches a global load for the ring, no register staging, and ONE block barrier per plane (the hand-over
// of the y-face fluxes, double-buffered) instead of three.
#define CD3_NP 6
__global__ void __launch_bounds__(3 * CD3_NT, 2) k_cd_tile3(FlowP P, CdT T, const float* __restrict__ u0, const float* __restrict__ mu0,
                                                           float* __restrict__ out, const DevScal* __restrict__ ds, int corrector,
                                                           const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1,
                                                           const __grid_constant__ CUtensorMap tm2)
{
    constexpr int ND = 3;
    extern __shared__ __align__(128) float4 cd_smem[];
    float* ring = reinterpret_cast<float*>(cd_smem);
    const Grid& g = P.g;
    const float dt = ds->dt;
    constexpr int SLOT = ND * CD3_PLANE;            // floats per ring slot (a multiple of 32: slots stay 128-byte aligned)
    float4* ex = reinterpret_cast<float4*>(ring + CD3_NP * SLOT);          // [2][ND][CD3_TY][CD_TX] lower-y-face fluxes
    const unsigned sring = (unsigned)__cvta_generic_to_shared(ring);
    const unsigned mbar = (unsigned)__cvta_generic_to_shared(ex + 2 * ND * CD3_NT);     // [CD3_NP] slot barriers
    const int comp = threadIdx.x / CD3_NT, t2 = threadIdx.x - comp * CD3_NT;
    const float Vi = ds->vel[comp];
    CdView2<CD3_TY> v;
    const int tx = t2 & (CD_TX - 1), ty = t2 / CD_TX;
    const int tofs = (ty + 2) * CD_W + 4 * (tx + 1);          // the thread's own group inside a plane
    const bool top = ty == CD3_TY - 1;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < CD3_NP; ++k) mbar_init(mbar + 8u * k, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned phases = 0;                           // parity of the next completion of each slot barrier
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        const int tix = tile % T.ntx, rem = tile / T.ntx;
        const int tiy = rem % T.nty, tiz = rem / T.nty;
        const int bx = 1 + 4 * CD_TX * tix, by = 1 + CD3_TY * tiy;
        const int z0 = 1 + T.zc * tiz, z1 = min(z0 + T.zc - 1, g.n[2]);
        const int gx = bx + 4 * tx, gy = by + ty;
        int nv = g.n[0] - gx + 1;
        nv = nv > 4 ? 4 : nv;
        if (gy > g.n[1]) nv = 0;
        // plane p of the tile (z0-2 <= p <= z1+2) lives in slot (p - z0 + 2) % CD3_NP
        auto issue = [&](int p, int slot) {
            const unsigned bar = mbar + 8u * (unsigned)slot, dst = sring + 4u * (unsigned)(slot * SLOT);
            const int cz = src_coord(p, g.n[2], g.per[2]);
            mbar_expect_tx(bar, (unsigned)(SLOT * 4));
            tma_box3(dst, &tm0, WL_OFF + bx - 4, by - 2, cz, bar);
            tma_box3(dst + 4u * CD3_PLANE, &tm1, WL_OFF + bx - 4, by - 2, cz, bar);
            tma_box3(dst + 8u * CD3_PLANE, &tm2, WL_OFF + bx - 4, by - 2, cz, bar);
        };
        auto arrived = [&](int slot) {
            mbar_wait(mbar + 8u * (unsigned)slot, (phases >> slot) & 1u);
            phases ^= 1u << slot;
        };
        __syncthreads();                           // the previous tile's reads are done (and the barriers are initialised)
        if (threadIdx.x == 0)
            for (int d = 0; d < CD3_NP && z0 - 2 + d <= z1 + 2; ++d) issue(z0 - 2 + d, d);
        for (int d = 0; d < 4; ++d) arrived(d);    // planes z0-2 .. z0+1; plane z+2 is awaited at the top of every step
        int s0 = 0;                                // ring slot of plane z-2
        float fz[4] = { 0.f, 0.f, 0.f, 0.f };      // flux through the upper z face of the previous plane
#pragma unroll 1
        for (int z = z0; z <= z1; ++z) {
            {
                int s = s0 + 4;
                if (s >= CD3_NP) s -= CD3_NP;
                arrived(s);                        // plane z+2
            }
#pragma unroll
            for (int d = 0; d < CD_NP; ++d) {
                int s = s0 + d;
                if (s >= CD3_NP) s -= CD3_NP;
                v.b[d] = ring + s * SLOT + tofs;
            }
            Cd2Part q;
            Cd2Pre pre;
            const bool first = z == z0;
            if (comp == 0)      { cd2_preload<ND, 0>(P, gx, gy, z, nv, u0, mu0, Vi, corrector, pre); cd2_fluxes<ND, 0>(P, v, gx, gy, z, top, first, fz, q); }
            else if (comp == 1) { cd2_preload<ND, 1>(P, gx, gy, z, nv, u0, mu0, Vi, corrector, pre); cd2_fluxes<ND, 1>(P, v, gx, gy, z, top, first, fz, q); }
            else                { cd2_preload<ND, 2>(P, gx, gy, z, nv, u0, mu0, Vi, corrector, pre); cd2_fluxes<ND, 2>(P, v, gx, gy, z, top, first, fz, q); }
            float4* exz = ex + (z & 1) * ND * CD3_NT;
            exz[(comp * CD3_TY + ty) * CD_TX + tx] = make_float4(q.fyl[0], q.fyl[1], q.fyl[2], q.fyl[3]);
            __syncthreads();                       // the lower-y-face fluxes of the plane are in shared memory; the ring reads of the plane are done
            if (threadIdx.x == 0 && z + 4 <= z1 + 2) issue(z + 4, s0);     // into the slot plane z-2 occupied; needed two steps from now
            float fyu[4];
            if (top) {
#pragma unroll
                for (int k = 0; k < 4; ++k) fyu[k] = q.fyu[k];
            } else {
                unpack4(exz[(comp * CD3_TY + ty + 1) * CD_TX + tx], fyu);
            }
            if (comp == 0)      cd2_output<ND, 0>(P, gx, gy, z, nv, q, fyu, pre, out, dt, corrector);
            else if (comp == 1) cd2_output<ND, 1>(P, gx, gy, z, nv, q, fyu, pre, out, dt, corrector);
            else                cd2_output<ND, 2>(P, gx, gy, z, nv, q, fyu, pre, out, dt, corrector);
            s0 = s0 + 1 == CD3_NP ? 0 : s0 + 1;
        }
    }
}

// ====================================================================== the band kernel
template <int ND, int I>
__device__ __forceinline__ void band_face(const FlowP& P, const float* __restrict__ w, const float* __restrict__ u0,
                                          const float* __restrict__ mu1, float* __restrict__ out, int c0, int c1, int c2,
                                          float dt, float Vi, float scale)
{
    const Grid& g = P.g;
    const int64_t id = gidx(g, c0, c1, c2);
    float acc = 0.0f;
    bool any = false;
#pragma unroll
    for (int j = 0; j < ND; ++j) {
        const float m1 = mu1[(I * ND + j) * g.nalloc + id];
        if (m1 == 0.0f) continue;
        int cp[3] = { c0, c1, c2 }, cm[3] = { c0, c1, c2 };
        cp[j] += 1; cm[j] -= 1;
        const float fp = f_at<ND, I>(P, w, u0, dt, Vi, cp[0], cp[1], cp[2]);
        const float fm = f_at<ND, I>(P, w, u0, dt, Vi, cm[0], cm[1], cm[2]);
        acc += m1 * 0.5f * (fp - fm);
        any = true;
    }
    if (any) out[I * g.nalloc + id] += scale * acc;
}

template <int ND>
__global__ void __launch_bounds__(128) k_cd_band(FlowP P, const float* __restrict__ w, const float* __restrict__ u0,
                                                 const float* __restrict__ mu1, float* __restrict__ out,
                                                 const DevScal* __restrict__ ds, const long long* __restrict__ list, int cap, int corrector)
{
    const Grid& g = P.g;
    const float dt = ds->dt;
    const float V[3] = { ds->vel[0], ds->vel[1], ds->vel[2] };
    const float scale = corrector ? 0.5f : 1.0f;
    // blockIdx.y = velocity component: the list holds one segment of cap / 3 entries per component (k_measure), so that a warp
    // runs ONE instantiation of band_face instead of up to three one after the other
    const int i = blockIdx.y, cap3 = cap / 3;
    const int cnt = ds->band_count[i];
    const bool fits = ds->band_count[0] <= cap3 && ds->band_count[1] <= cap3 && ds->band_count[2] <= cap3;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, t0 = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (fits) {
        for (int64_t e = t0; e < cnt; e += stride) {
            int64_t q = (list[(int64_t)i * cap3 + e] >> 2) - WL_OFF;
            const int c2 = ND == 3 ? (int)(q / g.sz) : 0;
            if (ND == 3) q -= (int64_t)c2 * g.sz;
            const int c1 = (int)(q / g.sy), c0 = (int)(q - (int64_t)c1 * g.sy);
            if (i == 0) band_face<ND, 0>(P, w, u0, mu1, out, c0, c1, c2, dt, V[0], scale);
            else if (i == 1) band_face<ND, 1>(P, w, u0, mu1, out, c0, c1, c2, dt, V[1], scale);
            else if (ND == 3) band_face<ND, 2>(P, w, u0, mu1, out, c0, c1, c2, dt, V[2], scale);
        }
    } else if (i == 0) {
        // the list overflowed (a body far larger than the capacity heuristic): scan every interior face
        const int64_t n01 = (int64_t)g.n[0] * g.n[1], tot = n01 * g.n[2];
        for (int64_t e = t0; e < tot; e += stride) {
            const int c2 = ND == 3 ? 1 + (int)(e / n01) : 0;
            const int64_t q = e % n01;
            const int c1 = 1 + (int)(q / g.n[0]), c0 = 1 + (int)(q % g.n[0]);
            band_face<ND, 0>(P, w, u0, mu1, out, c0, c1, c2, dt, V[0], scale);
            band_face<ND, 1>(P, w, u0, mu1, out, c0, c1, c2, dt, V[1], scale);
            if (ND == 3) band_face<ND, 2>(P, w, u0, mu1, out, c0, c1, c2, dt, V[2], scale);
        }
    }
}

// ====================================================================== host launcher
static CdT cd_tiling(const wl_sim* s, const Grid& g, int rows)
{
    CdT T;
    T.ntx = (g.n[0] + 4 * CD_TX - 1) / (4 * CD_TX);
    T.nty = (g.n[1] + rows - 1) / rows;
    T.zc = 1; T.ntz = 1;
    if (s->nd == 3) {
        // planes per tile: long marches amortise the four halo planes; keep >= ~6 tiles per resident block
        int zc = 32;
        while (zc > 8 && (int64_t)T.ntx * T.nty * ((g.n[2] + zc - 1) / zc) < (int64_t)s->sm_count * 12) zc /= 2;
        if (zc > g.n[2]) zc = g.n[2];
        T.zc = zc;
        T.ntz = (g.n[2] + zc - 1) / zc;
    }
    T.ntiles = T.ntx * T.nty * T.ntz;
    return T;
}

void wl_k_conv_diff_bdim(wl_sim* s, const float* w, const float* u0, float* out, int corrector)
{
    FlowP P = wl_flowp(s);
    const size_t smem2 = sizeof(float) * (size_t)(s->nd == 3 ? CD_NP : 1) * s->nd * CD_PLANE + sizeof(float4) * (size_t)s->nd * CD_NT;
    if (!(s->cd_attr_set & 2)) {
        cudaFuncSetAttribute(k_cd_tile2<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(float) * CD_NP * 3 * CD_PLANE + sizeof(float4) * 3 * CD_NT));
        cudaFuncSetAttribute(k_cd_tile2<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(float) * 2 * CD_PLANE + sizeof(float4) * 2 * CD_NT));
        s->cd_attr_set |= 2;
    }
    // the TMA-fed kernel where a box never has to wrap in x or y
    int cd3 = s->tma_cd && s->nd == 3 && !P.g.per[0] && !P.g.per[1];
    CUtensorMap tm[3];
    if (cd3)
        for (int c = 0; c < 3 && cd3; ++c) {
            const CUtensorMap* pm = wl_tensor_map_cached(s->tmc, w + c * P.g.nalloc, P.g, CD_W, CD3_R);
            cd3 = pm != nullptr;
            if (pm) tm[c] = *pm;
        }
    if (cd3) {
        const CdT T = cd_tiling(s, P.g, CD3_TY);
        const size_t smem3 = sizeof(float) * CD3_NP * 3 * CD3_PLANE + sizeof(float4) * 2 * 3 * CD3_NT + 8 * CD3_NP + 16;
        if (!(s->cd_attr_set & 4)) {
            cudaFuncSetAttribute(k_cd_tile3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem3);
            s->cd_attr_set |= 4;
        }
        ProfScope ps(s, WLK_CONVDIFF);
        k_cd_tile3<<<T.ntiles, 3 * CD3_NT, smem3, s->st>>>(P, T, u0, s->mu0, out, s->ds, corrector, tm[0], tm[1], tm[2]);
    } else {
        const CdT T = cd_tiling(s, P.g, CD2_TY);
        ProfScope ps(s, WLK_CONVDIFF);
        if (s->nd == 3) k_cd_tile2<3><<<T.ntiles, CD2_NT(3), smem2, s->st>>>(P, T, w, u0, s->mu0, out, s->ds, corrector);
        else            k_cd_tile2<2><<<T.ntiles, CD2_NT(2), smem2, s->st>>>(P, T, w, u0, s->mu0, out, s->ds, corrector);
    }
    if (s->cfg.body.kind != WL_BODY_NONE) {
        ProfScope ps(s, WLK_CONVDIFF_BAND);
        const int blocks = s->sm_count * 4;          // x the components (grid y)
        if (s->nd == 3) k_cd_band<3><<<dim3(blocks, 3), 128, 0, s->st>>>(P, w, u0, s->mu1, out, s->ds, s->band_list, s->band_cap, corrector);
        else            k_cd_band<2><<<dim3(blocks, 2), 128, 0, s->st>>>(P, w, u0, s->mu1, out, s->ds, s->band_list, s->band_cap, corrector);
    }
}
