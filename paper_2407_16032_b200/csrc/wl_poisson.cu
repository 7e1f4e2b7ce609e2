// wl_poisson.cu -- pressure projection: variable-coefficient Poisson problem solved by a
// geometric multigrid V-cycle with a Jacobi-preconditioned CG smoother (
// readings R-O, R-S, R-T of DESIGN.md).
//   (A x)_c = sum_i L[c+d_i,i](x[c+d_i]-x[c]) - L[c,i](x[c]-x[c-d_i]),  L = mu0 on level 0
// Periodic directions are handled by index wrap at load time: scalar level arrays keep no
// ghost values.  On non-periodic boundaries L = 0 on the boundary faces, so the (zero) ghost
// values never contribute.  Dot products stay on the device (PcgScal).
//
// Kernel shapes (wl_vec.cuh): float4 per thread along x, 256-thread blocks, z-marching with the
// z-neighbours in registers.  One PCG iteration is TWO passes over the level:
//   A: e' = beta e + iD r   (recomputed at the six neighbours instead of stored and re-read);
//      q = A e' ; gamma = q.e'                      [first iteration: e' = iD r, rho = r.e']
//   B: x += alpha e' ; r -= alpha q ; rho' = r.(iD r)
// z = iD r is never stored.  Tiles flagged "plain" (all face coefficients equal the level
// constant) skip the L and iD loads altogether.
#include <cstdio>
#include "wl_internal.h"
#include "wl_vec.cuh"

// ---------------------------------------------------------------- sources of a stencil operand
// A source returns the operand of the mat-vec at a float offset (scalar) or four of them.
template <bool PLAIN>
struct SrcFirst {                 // z = iD r
    const float* __restrict__ r; const float* __restrict__ iD; float iDc;
    __device__ __forceinline__ float s(int64_t i) const { return __fmul_rn(PLAIN ? iDc : __ldg(iD + i), __ldg(r + i)); }
    __device__ __forceinline__ float4 v(int64_t i) const
    {
        float4 a = ld4(r, i), d = PLAIN ? make_float4(iDc, iDc, iDc, iDc) : ld4(iD, i);
        return make_float4(__fmul_rn(d.x, a.x), __fmul_rn(d.y, a.y), __fmul_rn(d.z, a.z), __fmul_rn(d.w, a.w));
    }
};
template <bool PLAIN>
struct SrcNext {                  // beta e + iD r
    const float* __restrict__ e; const float* __restrict__ r; const float* __restrict__ iD; float beta, iDc;
    __device__ __forceinline__ float one(float ee, float rr, float dd) const { return __fmaf_rn(beta, ee, __fmul_rn(dd, rr)); }
    __device__ __forceinline__ float s(int64_t i) const { return one(__ldg(e + i), __ldg(r + i), PLAIN ? iDc : __ldg(iD + i)); }
    __device__ __forceinline__ float4 v(int64_t i) const
    {
        float4 a = ld4(e, i), b = ld4(r, i), d = PLAIN ? make_float4(iDc, iDc, iDc, iDc) : ld4(iD, i);
        return make_float4(one(a.x, b.x, d.x), one(a.y, b.y, d.y), one(a.z, b.z, d.z), one(a.w, b.w, d.w));
    }
};
struct SrcScaled {                // sc * p
    const float* __restrict__ p; float sc;
    __device__ __forceinline__ float s(int64_t i) const { return __fmul_rn(sc, __ldg(p + i)); }
    __device__ __forceinline__ float4 v(int64_t i) const
    {
        float4 a = ld4(p, i);
        return make_float4(__fmul_rn(sc, a.x), __fmul_rn(sc, a.y), __fmul_rn(sc, a.z), __fmul_rn(sc, a.w));
    }
};

// x-window of a row: w[0..5] = S(c0-1 .. c0+4), centre values given; periodic wrap in x.
template <class Src>
__device__ __forceinline__ void xwin(const Src& S, const Grid& g, int64_t row, int c0, const float (&cen)[4], float (&w)[6])
{
    const int n = g.n[0], per = g.per[0];
    w[1] = cen[0]; w[2] = cen[1]; w[3] = cen[2]; w[4] = cen[3];
    w[0] = S.s(row + ((c0 == 1 && per) ? n : c0 - 1));
    int ch = c0 + 4;
    if (ch > n + 1) ch = n + 1;                  // beyond the row: value unused
    if (ch == n + 1 && per) ch = 1;
    w[5] = S.s(row + ch);
    if (per && c0 + 3 > n) {                     // partial last group: cell n+1 lies inside the vector
        float first = S.s(row + 1);
#pragma unroll
        for (int k = 1; k <= 3; ++k) if (c0 + k == n + 1) w[k + 1] = first;
    }
}

// face coefficients of the thread's four cells on one plane
struct Coef { float x[5], y[4], yp[4], z[4], zp[4]; };

template <int ND, bool PLAIN>
__device__ __forceinline__ void coef_load(const Grid& g, const float* __restrict__ L, float Lc, int64_t i, Coef& C, bool first)
{
    if (PLAIN) {
#pragma unroll
        for (int k = 0; k < 4; ++k) { C.x[k] = Lc; C.y[k] = Lc; C.yp[k] = Lc; C.z[k] = Lc; C.zp[k] = Lc; }
        C.x[4] = Lc;
        return;
    }
    float4 a = ld4(L, i);
    C.x[0] = a.x; C.x[1] = a.y; C.x[2] = a.z; C.x[3] = a.w; C.x[4] = __ldg(L + i + 4);
    unpack4(ld4(L + g.nalloc, i), C.y);
    unpack4(ld4(L + g.nalloc, i + g.sy), C.yp);
    if (ND == 3) {
        if (first) unpack4(ld4(L + 2 * g.nalloc, i), C.z);
        else {
#pragma unroll
            for (int k = 0; k < 4; ++k) C.z[k] = C.zp[k];
        }
        unpack4(ld4(L + 2 * g.nalloc, i + g.sz), C.zp);
    }
}

template <int ND>
__device__ __forceinline__ float stencil(const Coef& C, int k, const float (&w)[6], const float (&ym)[4], const float (&yp)[4],
                                         const float (&zm)[4], const float (&zp)[4])
{
    const float ec = w[k + 1];
    float acc = 0.0f;
    acc += C.x[k + 1] * (w[k + 2] - ec) - C.x[k] * (ec - w[k]);
    acc += C.yp[k] * (yp[k] - ec) - C.y[k] * (ec - ym[k]);
    if (ND == 3) acc += C.zp[k] * (zp[k] - ec) - C.z[k] * (ec - zm[k]);
    return acc;
}

// Marches one tile: for every plane calls F(z, idx, w, q[4]) with w = x-window of the operand and
// q = A operand at the thread's four cells.
template <int ND, bool PLAIN, class Src, class Fn>
__device__ __forceinline__ void march(const Grid& g, const VPos& p, const Src& S, const float* __restrict__ L, float Lc, Fn&& F)
{
    const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy;
    const int64_t rm = (int64_t)WL_OFF + (int64_t)nb_lo(p.c1, g.n[1], g.per[1]) * g.sy;
    const int64_t rp = (int64_t)WL_OFF + (int64_t)nb_hi(p.c1, g.n[1], g.per[1]) * g.sy;
    float zm[4] = { 0.f, 0.f, 0.f, 0.f }, zc[4], zp[4] = { 0.f, 0.f, 0.f, 0.f };
    if (ND == 3) unpack4(S.v(rc + p.c0 + (int64_t)nb_lo(p.z0, g.n[2], g.per[2]) * g.sz), zm);
    unpack4(S.v(rc + p.c0 + (int64_t)p.z0 * g.sz), zc);
    Coef C;
    for (int z = p.z0; z <= p.z1; ++z) {
        const int64_t zo = (int64_t)z * g.sz;
        float w[6], ym[4], yp[4];
        xwin(S, g, rc + zo, p.c0, zc, w);
        unpack4(S.v(rm + zo + p.c0), ym);
        unpack4(S.v(rp + zo + p.c0), yp);
        if (ND == 3) unpack4(S.v(rc + p.c0 + (int64_t)nb_hi(z, g.n[2], g.per[2]) * g.sz), zp);
        coef_load<ND, PLAIN>(g, L, Lc, rc + zo + p.c0, C, z == p.z0);
        float q[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) q[k] = stencil<ND>(C, k, w, ym, yp, zm, zp);
        F(z, rc + zo + p.c0, w, q);
        if (ND == 3) {
#pragma unroll
            for (int k = 0; k < 4; ++k) { zm[k] = zc[k]; zc[k] = zp[k]; }
        }
    }
}

// ---------------------------------------------------------------- diagonal + plain flags
// D = -sum_i (L[c,i] + L[c+d_i,i]); iD = 1/D if |D| > 2n*1e-6 else 0 (R-O).  A tile is plain
// when all 2n face coefficients of all of its cells equal Lc.
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_diag_flags(Grid g, VT vt, const float* __restrict__ L, float Lc, float* __restrict__ iD, int* __restrict__ plain)
{
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        int ok = 1;
        if (p.nv > 0) {
            const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy;
            Coef C;
            for (int z = p.z0; z <= p.z1; ++z) {
                const int64_t i = rc + (int64_t)z * g.sz + p.c0;
                coef_load<ND, false>(g, L, Lc, i, C, z == p.z0);
                float d[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float D = 0.0f;
                    D -= C.x[k] + C.x[k + 1];
                    D -= C.y[k] + C.yp[k];
                    if (ND == 3) D -= C.z[k] + C.zp[k];
                    d[k] = fabsf(D) > 2.0f * ND * 1e-6f ? 1.0f / D : 0.0f;
                    if (k < p.nv) {
                        bool same = C.x[k] == Lc && C.x[k + 1] == Lc && C.y[k] == Lc && C.yp[k] == Lc;
                        if (ND == 3) same = same && C.z[k] == Lc && C.zp[k] == Lc;
                        if (!same) ok = 0;
                    }
                }
                st4(iD, i, d, p.nv);
            }
        }
        ok = __syncthreads_and(ok);
        if (threadIdx.x == 0) plain[tile] = ok;
    }
}

// The PCG pass A recomputes e' = beta e + iD r at the six neighbours of every cell, so a tile may
// only use the constant iDc if the cells one step outside it are uniform too: a tile is plain
// when it and its face-neighbour tiles (periodic wrap) are uniform.  A missing neighbour means a
// domain boundary, and boundary tiles are never uniform (L = 0 on the boundary faces).
__global__ void k_plain_dilate(VT vt, int per0, int per1, int per2, const int* __restrict__ self, int* __restrict__ plain)
{
    for (int tile = blockIdx.x * blockDim.x + threadIdx.x; tile < vt.ntiles; tile += gridDim.x * blockDim.x) {
        int t[3] = { tile % vt.ntx, (tile / vt.ntx) % vt.nty, tile / (vt.ntx * vt.nty) };
        const int nt[3] = { vt.ntx, vt.nty, vt.ntz };
        const int per[3] = { per0, per1, per2 };
        int ok = self[tile];
        for (int d = 0; d < 3 && ok; ++d)
            for (int s = -1; s <= 1; s += 2) {
                int q[3] = { t[0], t[1], t[2] };
                q[d] += s;
                if (q[d] < 0 || q[d] >= nt[d]) {
                    if (!per[d]) continue;
                    q[d] = q[d] < 0 ? nt[d] - 1 : 0;
                }
                ok = ok && self[q[0] + vt.ntx * (q[1] + vt.nty * q[2])];
            }
        plain[tile] = ok;
    }
}

// ---- coefficient restriction (R-S): coarse face coefficient = 1/2 * sum of the 2^(n-1) fine
// face coefficients on that coarse face.  One thread per coarse cell C, faces C_i = 1..n_i+1
// (the extra upper plane is covered by letting C_i run to n_i+1 for component i).
template <int ND>
__global__ void __launch_bounds__(512) k_restrict_L(Grid gf, Grid gc, Tiling T, const float* __restrict__ Lf, float* __restrict__ Lc)
{
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int C[3];
        if (!tile_cell(T, tile, C[0], C[1], C[2])) continue;
        int64_t idc = gidx(gc, C[0], C[1], C[2]);
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            // component i needs the other coordinates interior
            bool ok = true;
#pragma unroll
            for (int d = 0; d < ND; ++d) if (d != i && C[d] > gc.n[d]) ok = false;
            if (!ok) continue;
            int b[3] = { 2 * C[0] - 1, 2 * C[1] - 1, ND == 3 ? 2 * C[2] - 1 : 0 };
            float sum = 0.0f;
            const int n1 = 2, n2 = ND == 3 ? 2 : 1;
            for (int a2 = 0; a2 < n2; ++a2)
                for (int a1 = 0; a1 < n1; ++a1)
                    for (int a0 = 0; a0 < 2; ++a0) {
                        int a[3] = { a0, a1, a2 };
                        if (a[i] != 0) continue;
                        sum += Lf[i * gf.nalloc + gidx(gf, b[0] + a0, b[1] + a1, b[2] + a2)];
                    }
            Lc[i * gc.nalloc + idc] = 0.5f * sum;
        }
    }
}

// ---------------------------------------------------------------- project!, first half
// (R-K): pscale = w dt; x = pscale p; r = div u - A x.
template <int ND, bool PLAIN>
__device__ __forceinline__ void residual_tile(const Grid& g, const VPos& p, const float* __restrict__ u, const float* __restrict__ L, float Lc,
                                              const float* __restrict__ pr, float sc, float* __restrict__ x, float* __restrict__ r)
{
    SrcScaled S{ pr, sc };
    float uzc[4] = { 0.f, 0.f, 0.f, 0.f };
    if (ND == 3) unpack4(ld4(u + 2 * g.nalloc, (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + (int64_t)p.z0 * g.sz + p.c0), uzc);
    march<ND, PLAIN>(g, p, S, L, Lc, [&](int z, int64_t i, const float (&w)[6], const float (&q)[4]) {
        // u ghosts are BC-filled: plain +1 neighbours
        float ux[4], uy[4], uyp[4], uzp[4] = { 0.f, 0.f, 0.f, 0.f }, xo[4], ro[4];
        unpack4(ld4(u, i), ux);
        const float ux4 = __ldg(u + i + 4);
        unpack4(ld4(u + g.nalloc, i), uy);
        unpack4(ld4(u + g.nalloc, i + g.sy), uyp);
        if (ND == 3) unpack4(ld4(u + 2 * g.nalloc, i + g.sz), uzp);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            float div = 0.0f;
            div += (k < 3 ? ux[k + 1] : ux4) - ux[k];
            div += uyp[k] - uy[k];
            if (ND == 3) div += uzp[k] - uzc[k];
            xo[k] = w[k + 1];
            ro[k] = div - q[k];
            if (ND == 3) uzc[k] = uzp[k];
        }
        st4(x, i, xo, p.nv);
        st4(r, i, ro, p.nv);
    });
}

template <int ND>
__global__ void __launch_bounds__(WL_VB) k_residual(Grid g, VT vt, const int* __restrict__ plain, const float* __restrict__ u, const float* __restrict__ L, float Lc,
                                                    const float* __restrict__ p, float* __restrict__ x, float* __restrict__ r, DevScal* ds, float w)
{
    const float sc = w * ds->dt;
    if (blockIdx.x == 0 && threadIdx.x == 0) ds->pscale = sc;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos ps = vt_pos(g, vt, tile);
        if (ps.nv == 0) continue;
        if (plain[tile]) residual_tile<ND, true>(g, ps, u, L, Lc, p, sc, x, r);
        else             residual_tile<ND, false>(g, ps, u, L, Lc, p, sc, x, r);
    }
}

// ---------------------------------------------------------------- project!, second half
// (P:88 kernel): u[c,i] -= L[c,i] (x[c] - x[c-d_i]); p = x / pscale
template <int ND, bool PLAIN>
__device__ __forceinline__ void gradient_tile(const Grid& g, const VPos& p, float* __restrict__ u, const float* __restrict__ L, float Lc,
                                              const float* __restrict__ x, float* __restrict__ pr, float isc)
{
    const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy;
    const int64_t rm = (int64_t)WL_OFF + (int64_t)nb_lo(p.c1, g.n[1], g.per[1]) * g.sy;
    float zm[4] = { 0.f, 0.f, 0.f, 0.f };
    if (ND == 3) unpack4(ld4(x, rc + p.c0 + (int64_t)nb_lo(p.z0, g.n[2], g.per[2]) * g.sz), zm);
    for (int z = p.z0; z <= p.z1; ++z) {
        const int64_t i = rc + (int64_t)z * g.sz + p.c0;
        float xc[4], ym[4], o[4];
        unpack4(ld4(x, i), xc);
        const float xm = __ldg(x + rc + (int64_t)z * g.sz + ((p.c0 == 1 && g.per[0]) ? g.n[0] : p.c0 - 1));
        unpack4(ld4(x, rm + (int64_t)z * g.sz + p.c0), ym);
        float l[4] = { Lc, Lc, Lc, Lc }, uu[4];
        // x component
        if (!PLAIN) unpack4(ld4(L, i), l);
        unpack4(*reinterpret_cast<const float4*>(u + i), uu);
#pragma unroll
        for (int k = 0; k < 4; ++k) o[k] = uu[k] - l[k] * (xc[k] - (k == 0 ? xm : xc[k - 1]));
        st4(u, i, o, p.nv);
        // y component
        if (!PLAIN) unpack4(ld4(L + g.nalloc, i), l);
        unpack4(*reinterpret_cast<const float4*>(u + g.nalloc + i), uu);
#pragma unroll
        for (int k = 0; k < 4; ++k) o[k] = uu[k] - l[k] * (xc[k] - ym[k]);
        st4(u + g.nalloc, i, o, p.nv);
        if (ND == 3) {
            if (!PLAIN) unpack4(ld4(L + 2 * g.nalloc, i), l);
            unpack4(*reinterpret_cast<const float4*>(u + 2 * g.nalloc + i), uu);
#pragma unroll
            for (int k = 0; k < 4; ++k) { o[k] = uu[k] - l[k] * (xc[k] - zm[k]); zm[k] = xc[k]; }
            st4(u + 2 * g.nalloc, i, o, p.nv);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) o[k] = xc[k] * isc;
        st4(pr, i, o, p.nv);
    }
}

template <int ND>
__global__ void __launch_bounds__(WL_VB) k_apply_gradient(Grid g, VT vt, const int* __restrict__ plain, float* __restrict__ u, const float* __restrict__ L, float Lc,
                                                          const float* __restrict__ x, float* __restrict__ p, const DevScal* __restrict__ ds)
{
    const float isc = 1.0f / ds->pscale;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos ps = vt_pos(g, vt, tile);
        if (ps.nv == 0) continue;
        if (plain[tile]) gradient_tile<ND, true>(g, ps, u, L, Lc, x, p, isc);
        else             gradient_tile<ND, false>(g, ps, u, L, Lc, x, p, isc);
    }
}

// ---------------------------------------------------------------- residual restriction
// r_c[C] = sum of the 2^n children; x_c = 0 (R-S).  One thread per four coarse cells.
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_restrict_r(Grid gf, Grid gc, VT vt, const float* __restrict__ rf, float* __restrict__ rc, float* __restrict__ xc)
{
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(gc, vt, tile);
        if (p.nv == 0) continue;
        const int f0 = 2 * p.c0 - 1, f1 = 2 * p.c1 - 1;      // first fine child (f0 = 1 + 8 gx: 32-byte aligned)
        for (int z = p.z0; z <= p.z1; ++z) {
            float s[4] = { 0.f, 0.f, 0.f, 0.f };
            const int nz = ND == 3 ? 2 : 1;
            for (int a2 = 0; a2 < nz; ++a2)
                for (int a1 = 0; a1 < 2; ++a1) {
                    const int64_t b = gidx(gf, f0, f1 + a1, ND == 3 ? 2 * z - 1 + a2 : 0);
                    float4 lo = ld4(rf, b);
                    s[0] += lo.x; s[0] += lo.y; s[1] += lo.z; s[1] += lo.w;
                    if (p.nv > 2) {
                        float4 hi = ld4(rf, b + 4);
                        s[2] += hi.x; s[2] += hi.y; s[3] += hi.z; s[3] += hi.w;
                    }
                }
            const int64_t i = gidx(gc, p.c0, p.c1, z);
            const float zero[4] = { 0.f, 0.f, 0.f, 0.f };
            st4(rc, i, s, p.nv);
            st4(xc, i, zero, p.nv);
        }
    }
}

// ---------------------------------------------------------------- prolongation + increment
// e = P x_c (piecewise constant); x_f += e; r_f -= A_f e (R-S)
__device__ __forceinline__ int par(int c) { return (c + 1) >> 1; }          // parent of a fine index (ghost 0 -> 0, n+1 -> n/2+1)
__device__ __forceinline__ int wrapC(int C, int n, int per) { if (per) { if (C < 1) C += n; else if (C > n) C -= n; } return C; }

template <int ND, bool PLAIN>
__device__ __forceinline__ void prolong_tile(const Grid& gf, const Grid& gc, const VPos& p, const float* __restrict__ L, float Lc,
                                             const float* __restrict__ xc, float* __restrict__ xf, float* __restrict__ rf)
{
    const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * gf.sy;
    const int Ca = par(p.c0);                       // parents of the group: Ca, Ca, Ca+1, Ca+1
    const int X0 = wrapC(Ca - 1, gc.n[0], gc.per[0]), X1 = wrapC(Ca, gc.n[0], gc.per[0]);
    const int X2 = wrapC(Ca + 1, gc.n[0], gc.per[0]), X3 = wrapC(Ca + 2, gc.n[0], gc.per[0]);
    const int Y = par(p.c1);
    const int Ym = par(nb_lo(p.c1, gf.n[1], gf.per[1])), Yp = par(nb_hi(p.c1, gf.n[1], gf.per[1]));
    Coef C;
    for (int z = p.z0; z <= p.z1; ++z) {
        const int64_t i = rc + (int64_t)z * gf.sz + p.c0;
        const int Z = ND == 3 ? par(z) : 0;
        const int64_t row = gidx(gc, 0, Y, Z);
        const float v0 = __ldg(xc + row + X0), v1 = __ldg(xc + row + X1), v2 = __ldg(xc + row + X2), v3 = __ldg(xc + row + X3);
        const float w[6] = { v0, v1, v1, v2, v2, v3 };
        float ym[4], yp[4], zm[4] = { 0.f, 0.f, 0.f, 0.f }, zp[4] = { 0.f, 0.f, 0.f, 0.f };
        {
            const int64_t a = gidx(gc, 0, Ym, Z), b = gidx(gc, 0, Yp, Z);
            float a1 = __ldg(xc + a + X1), a2 = __ldg(xc + a + X2), b1 = __ldg(xc + b + X1), b2 = __ldg(xc + b + X2);
            ym[0] = a1; ym[1] = a1; ym[2] = a2; ym[3] = a2;
            yp[0] = b1; yp[1] = b1; yp[2] = b2; yp[3] = b2;
        }
        if (ND == 3) {
            const int64_t a = gidx(gc, 0, Y, par(nb_lo(z, gf.n[2], gf.per[2]))), b = gidx(gc, 0, Y, par(nb_hi(z, gf.n[2], gf.per[2])));
            float a1 = __ldg(xc + a + X1), a2 = __ldg(xc + a + X2), b1 = __ldg(xc + b + X1), b2 = __ldg(xc + b + X2);
            zm[0] = a1; zm[1] = a1; zm[2] = a2; zm[3] = a2;
            zp[0] = b1; zp[1] = b1; zp[2] = b2; zp[3] = b2;
        }
        coef_load<ND, PLAIN>(gf, L, Lc, i, C, z == p.z0);
        float xo[4], ro[4];
        unpack4(*reinterpret_cast<const float4*>(xf + i), xo);
        unpack4(*reinterpret_cast<const float4*>(rf + i), ro);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            xo[k] += w[k + 1];
            ro[k] -= stencil<ND>(C, k, w, ym, yp, zm, zp);
        }
        st4(xf, i, xo, p.nv);
        st4(rf, i, ro, p.nv);
    }
}

template <int ND>
__global__ void __launch_bounds__(WL_VB) k_prolong(Grid gf, Grid gc, VT vt, const int* __restrict__ plain, const float* __restrict__ L, float Lc,
                                                   const float* __restrict__ xc, float* __restrict__ xf, float* __restrict__ rf)
{
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(gf, vt, tile);
        if (p.nv == 0) continue;
        if (plain[tile]) prolong_tile<ND, true>(gf, gc, p, L, Lc, xc, xf, rf);
        else             prolong_tile<ND, false>(gf, gc, p, L, Lc, xc, xf, rf);
    }
}

// ---------------------------------------------------------------- Jacobi-PCG smoother
// (R-S, R-T), restarted at every call:
//   z = e = iD r; rho = r.z; if |rho| < tau return
//   loop k = 1..it: q = A e; gamma = q.e; alpha = rho/gamma; x += alpha e; r -= alpha q;
//                   if k == it break; z = iD r; rho' = r.z; if |rho'| < tau or < theta |rho0| break;
//                   beta = rho'/rho; e = beta e + z; rho = rho'
template <int ND, int FIRST, bool PLAIN>
__device__ __forceinline__ void pcgA_tile(const Grid& g, const VPos& p, const float* __restrict__ L, float Lc, float iDc,
                                          const float* __restrict__ ein, const float* __restrict__ r, const float* __restrict__ iD, float beta,
                                          float* __restrict__ eout, float* __restrict__ q, double& gam, double& rho)
{
    auto body = [&](int z, int64_t i, const float (&w)[6], const float (&qq)[4]) {
        float eo[4] = { w[1], w[2], w[3], w[4] };
        st4(eout, i, eo, p.nv);
        st4(q, i, qq, p.nv);
        float rr[4] = { 0.f, 0.f, 0.f, 0.f };
        if (FIRST) unpack4(ld4(r, i), rr);
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (k < p.nv) {
                gam += (double)qq[k] * (double)eo[k];
                if (FIRST) rho += (double)eo[k] * (double)rr[k];
            }
    };
    if (FIRST) { SrcFirst<PLAIN> S{ r, iD, iDc }; march<ND, PLAIN>(g, p, S, L, Lc, body); }
    else       { SrcNext<PLAIN> S{ ein, r, iD, beta, iDc }; march<ND, PLAIN>(g, p, S, L, Lc, body); }
}

template <int ND, int FIRST>
__global__ void __launch_bounds__(WL_VB) k_pcg_A(Grid g, VT vt, const int* __restrict__ plain, const float* __restrict__ L, float Lc, float iDc,
                                                 const float* __restrict__ ein, const float* __restrict__ r, const float* __restrict__ iD,
                                                 float* __restrict__ eout, float* __restrict__ q, PcgScal* sc, RedBuf rb)
{
    if (!FIRST && !sc->live) return;          // uniform across the grid: written by an earlier kernel
    const float beta = FIRST ? 0.0f : (float)sc->beta;
    double v[2] = { 0.0, 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
        if (plain[tile]) pcgA_tile<ND, FIRST, true>(g, p, L, Lc, iDc, ein, r, iD, beta, eout, q, v[0], v[1]);
        else             pcgA_tile<ND, FIRST, false>(g, p, L, Lc, iDc, ein, r, iD, beta, eout, q, v[0], v[1]);
    }
    if (grid_reduce<2, OpSum>(v, rb)) {
        if (threadIdx.x == 0) {
            double gamma = v[0];
            int live = 1;
            if (FIRST) {
                sc->rho = v[1]; sc->rho0 = v[1]; sc->beta = 0.0;
                live = fabs(v[1]) < WL_TAU ? 0 : 1;
            }
            sc->gamma = gamma;
            if (gamma == 0.0 || !isfinite(gamma) || !live) { sc->live = 0; sc->alpha = 0.0; }
            else { sc->live = 1; sc->alpha = sc->rho / gamma; }
        }
    }
}

// x += alpha e; r -= alpha q; unless last: rho' = r.(iD r) -> beta
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_pcg_B(Grid g, VT vt, const int* __restrict__ plain, float iDc, float* __restrict__ x, float* __restrict__ r,
                                                 const float* __restrict__ e, const float* __restrict__ q, const float* __restrict__ iD,
                                                 PcgScal* sc, RedBuf rb, int last)
{
    if (!sc->live) return;
    const float alpha = (float)sc->alpha;
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
        const bool pl = plain[tile] != 0;
        const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + p.c0;
        for (int z = p.z0; z <= p.z1; ++z) {
            const int64_t i = rc + (int64_t)z * g.sz;
            float xo[4], ro[4], ee[4], qq[4], dd[4] = { iDc, iDc, iDc, iDc };
            unpack4(*reinterpret_cast<const float4*>(x + i), xo);
            unpack4(*reinterpret_cast<const float4*>(r + i), ro);
            unpack4(ld4(e, i), ee);
            unpack4(ld4(q, i), qq);
            if (!last && !pl) unpack4(ld4(iD, i), dd);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                xo[k] += alpha * ee[k];
                ro[k] -= alpha * qq[k];
                if (!last && k < p.nv) {
                    float zz = __fmul_rn(dd[k], ro[k]);
                    v[0] += (double)zz * (double)ro[k];
                }
            }
            st4(x, i, xo, p.nv);
            st4(r, i, ro, p.nv);
        }
    }
    if (last) return;
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) {
            double rho2 = v[0];
            if (fabs(rho2) < WL_TAU || fabs(rho2) < WL_THETA * fabs(sc->rho0)) sc->live = 0;
            else { sc->beta = rho2 / sc->rho; sc->rho = rho2; }
        }
    }
}

template <int ND>
__global__ void __launch_bounds__(512) k_resmax(Grid g, Tiling T, const float* __restrict__ r, DevScal* ds, RedBuf rb)
{
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        double a = fabs((double)r[gidx(g, c0, c1, c2)]);
        if (a > v[0] || a != a) v[0] = a;
    }
    if (grid_reduce<1, OpMax>(v, rb)) {
        if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) ds->resmax = v[0];
    }
}

// ================================================================== host launchers
#define DISPATCH(s, cls, coarse, kern, T, ...)                                               \
    do {                                                                                     \
        ProfScope ps_(s, cls, coarse);                                                       \
        if ((s)->nd == 3) kern<3><<<wl_grid(s, T), wl_block(3), 0, (s)->st>>>(__VA_ARGS__);  \
        else              kern<2><<<wl_grid(s, T), wl_block(2), 0, (s)->st>>>(__VA_ARGS__);  \
    } while (0)

// vector-tile kernels: 256-thread blocks, persistent grid
#define VDISPATCH(s, cls, coarse, vt, kern2, kern3, ...)                                     \
    do {                                                                                     \
        ProfScope ps_(s, cls, coarse);                                                       \
        if ((s)->nd == 3) kern3<<<wl_vgrid(s, vt), WL_VB, 0, (s)->st>>>(__VA_ARGS__);        \
        else              kern2<<<wl_vgrid(s, vt), WL_VB, 0, (s)->st>>>(__VA_ARGS__);        \
    } while (0)

void wl_k_poisson_update(wl_sim* s)
{
    for (int l = 0; l < s->nlev; ++l) {
        Level& lv = s->lev[l];
        if (l > 0) {
            Level& lf = s->lev[l - 1];
            int o[3] = { 1, 1, s->nd == 3 ? 1 : 0 };
            int e[3] = { lv.g.n[0] + 1, lv.g.n[1] + 1, s->nd == 3 ? lv.g.n[2] + 1 : 1 };
            Tiling T = wl_tiling(s->nd, o, e);
            DISPATCH(s, WLK_POISSON_UPDATE, l > 1, k_restrict_L, T, lf.g, lv.g, T, lf.L, lv.L);
        }
        VDISPATCH(s, WLK_POISSON_UPDATE, l > 0, lv.vt, k_diag_flags<2>, k_diag_flags<3>, lv.g, lv.vt, lv.L, lv.Lc, lv.iD, lv.uniform);
        {
            ProfScope ps_(s, WLK_POISSON_UPDATE, l > 0);
            int nb = (lv.vt.ntiles + 255) / 256;
            k_plain_dilate<<<nb < 64 ? nb : 64, 256, 0, s->st>>>(lv.vt, lv.g.per[0], lv.g.per[1], lv.g.per[2], lv.uniform, lv.plain);
        }
    }
}

void wl_k_residual(wl_sim* s, const float* u, float w)
{
    Level& lv = s->lev[0];
    VDISPATCH(s, WLK_RESIDUAL, 0, lv.vt, k_residual<2>, k_residual<3>, lv.g, lv.vt, lv.plain, u, lv.L, lv.Lc, s->p, lv.x, lv.r, s->ds, w);
}

void wl_k_apply_gradient(wl_sim* s, float* u)
{
    Level& lv = s->lev[0];
    VDISPATCH(s, WLK_GRADIENT, 0, lv.vt, k_apply_gradient<2>, k_apply_gradient<3>, lv.g, lv.vt, lv.plain, u, lv.L, lv.Lc, lv.x, s->p, s->ds);
}

void wl_k_restrict(wl_sim* s, int l)
{
    Level &lf = s->lev[l], &lc = s->lev[l + 1];
    VDISPATCH(s, WLK_RESTRICT, l > 0, lc.vt, k_restrict_r<2>, k_restrict_r<3>, lf.g, lc.g, lc.vt, lf.r, lc.r, lc.x);
}

void wl_k_prolong(wl_sim* s, int l)
{
    Level &lf = s->lev[l], &lc = s->lev[l + 1];
    VDISPATCH(s, WLK_PROLONG, l > 0, lf.vt, k_prolong<2>, k_prolong<3>, lf.g, lc.g, lf.vt, lf.plain, lf.L, lf.Lc, lc.x, lf.x, lf.r);
}

void wl_k_smooth(wl_sim* s, int l, int iters)
{
    Level& lv = s->lev[l];
    PcgScal* sc = &s->ds->pcg[l];
    float* ea = lv.e;      // direction written by the running A pass
    float* eb = lv.e2;     // previous direction
    for (int k = 1; k <= iters; ++k) {
        if (k == 1)
            VDISPATCH(s, WLK_PCG_MATVEC, l > 0, lv.vt, (k_pcg_A<2, 1>), (k_pcg_A<3, 1>), lv.g, lv.vt, lv.plain, lv.L, lv.Lc, lv.iDc,
                      eb, lv.r, lv.iD, ea, lv.q, sc, s->rb);
        else
            VDISPATCH(s, WLK_PCG_MATVEC, l > 0, lv.vt, (k_pcg_A<2, 0>), (k_pcg_A<3, 0>), lv.g, lv.vt, lv.plain, lv.L, lv.Lc, lv.iDc,
                      eb, lv.r, lv.iD, ea, lv.q, sc, s->rb);
        VDISPATCH(s, WLK_PCG_UPDATE, l > 0, lv.vt, k_pcg_B<2>, k_pcg_B<3>, lv.g, lv.vt, lv.plain, lv.iDc, lv.x, lv.r, ea, lv.q, lv.iD, sc, s->rb,
                  k == iters ? 1 : 0);
        float* t = ea; ea = eb; eb = t;
    }
}

void wl_k_vcycle(wl_sim* s, int l)
{
    if (l + 1 >= s->nlev) return;
    wl_k_restrict(s, l);
    if (l + 1 < s->nlev - 1) wl_k_vcycle(s, l + 1);
    wl_k_smooth(s, l + 1, s->cfg.mg.smooth_iters);
    wl_k_prolong(s, l);
}

void wl_k_resmax(wl_sim* s)
{
    Level& lv = s->lev[0];
    Tiling T = wl_tiles_interior(s, lv.g);
    DISPATCH(s, WLK_RESMAX, 0, k_resmax, T, lv.g, T, lv.r, s->ds, s->rb);
}
