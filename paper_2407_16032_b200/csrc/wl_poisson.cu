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
//      q = A e' ; gamma = q.e'       [first iteration: e' = iD (r - m), rho = (r - m).e'; R-T2]
//   B: x += alpha e' ; r -= alpha q ; rho' = r.(iD r)
// z = iD r is never stored.  Every tile carries a mode (wl_vec.cuh): TM_GEN loads L and iD, the
// uniform modes TM_PLB / TM_PLI take them from the cell position / as constants.  On 3-D levels
// pass A runs in wl_pcgfast.cu (shared memory, TMA); k_pcg_A here serves 2-D and ragged levels and
// the persistent kernels.  Levels of at most 1 M cells run as chains of passes inside k_coarse
// (cooperative launch, grid barrier between passes); the small ones on chip in k_small (wl_small.cu, one thread-block cluster).
#include <cstdio>
#include <cstdlib>
#include "wl_internal.h"
#include "wl_vec.cuh"
#include <cooperative_groups.h>

// minimum resident blocks per SM the register allocation aims at (tuned on B200, profiles/)
#ifndef WL_A_MINB
#define WL_A_MINB 2
#endif
#ifndef WL_B_MINB
#define WL_B_MINB 4
#endif
#ifndef WL_PK_SLOT
#define WL_PK_SLOT 4      // doubles per block slot of the k_coarse partial sums: one 32-byte sector each
#endif
#ifndef WL_G_MINB
#define WL_G_MINB 4
#endif
#ifndef WL_R_MINB
#define WL_R_MINB 2
#endif
#ifndef WL_P_MINB
#define WL_P_MINB 4
#endif
#ifndef WL_PK_MINB
#define WL_PK_MINB 2
#endif

// Position bookkeeping of one thread of a TM_PLB tile.  iD of a body-free cell with k boundary
// faces is 1/(-(2 ND - k) Lc): the same correctly rounded quotient k_diag_flags stores.
template <int ND>
struct Ana {
    float Lc, tab[4];
    int xm;        // bit k (k = 0..5): cell c0-1+k has a non-periodic boundary x-face
    int by[3];     // rows c1-1, c1, c1+1 have a non-periodic boundary y-face
    __device__ __forceinline__ void init(const Grid& g, float Lc_, const VPos& p)
    {
        Lc = Lc_;
#pragma unroll
        for (int k = 0; k < 4; ++k) tab[k] = 1.0f / (-(float)(2 * ND - k) * Lc_);
        xm = 0;
        if (!g.per[0]) {
#pragma unroll
            for (int k = 0; k < 6; ++k) { const int c = p.c0 - 1 + k; if (c == 1 || c == g.n[0]) xm |= 1 << k; }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) { const int c = p.c1 - 1 + k; by[k] = (!g.per[1] && (c == 1 || c == g.n[1])) ? 1 : 0; }
    }
    __device__ __forceinline__ int bz(const Grid& g, int z) const { return (ND == 3 && !g.per[2] && (z == 1 || z == g.n[2])) ? 1 : 0; }
    __device__ __forceinline__ float pick(int n) const { return n == 0 ? tab[0] : (n == 1 ? tab[1] : (n == 2 ? tab[2] : tab[3])); }
};

// inverse diagonal at a float4 group of the thread's column (cnt = boundary faces in y and z of that
// row / plane) or at one of the two window ends (window position k = 0 or 5)
template <int ND, int MODE>
struct IDiag {
    const float* iD; float iDc; const Ana<ND>* a;
    __device__ __forceinline__ float4 v(int64_t i, int cnt) const
    {
        if (MODE == TM_GEN) return ld4(iD, i);
        if (MODE == TM_PLI) return make_float4(iDc, iDc, iDc, iDc);
        const float b = a->pick(cnt), c = a->pick(cnt + 1);
        const int xm = a->xm;
        return make_float4((xm & 2) ? c : b, (xm & 4) ? c : b, (xm & 8) ? c : b, (xm & 16) ? c : b);
    }
    __device__ __forceinline__ float s(int64_t i, int cnt, int k) const
    {
        if (MODE == TM_GEN) return ld1(iD, i);
        if (MODE == TM_PLI) return iDc;
        return a->pick(cnt + ((a->xm >> k) & 1));
    }
};

// ---------------------------------------------------------------- sources of a stencil operand
// A source returns the operand of the mat-vec at a float offset (scalar) or four of them.
template <int ND, int MODE>
struct SrcFirst {                 // z = iD (r - m), m = mean of r over the coupled cells (R-T2)
    const float* r; IDiag<ND, MODE> D; float m;
    __device__ __forceinline__ float s(int64_t i, int cnt, int k) const { return __fmul_rn(D.s(i, cnt, k), ld1(r, i) - m); }
    __device__ __forceinline__ float4 v(int64_t i, int cnt) const
    {
        const float4 a = ld4(r, i), d = D.v(i, cnt);
        return make_float4(__fmul_rn(d.x, a.x - m), __fmul_rn(d.y, a.y - m), __fmul_rn(d.z, a.z - m), __fmul_rn(d.w, a.w - m));
    }
};
template <int ND, int MODE>
struct SrcNext {                  // beta e + iD r
    const float* e; const float* r; IDiag<ND, MODE> D; float beta;
    __device__ __forceinline__ float one(float ee, float rr, float dd) const { return __fmaf_rn(beta, ee, __fmul_rn(dd, rr)); }
    __device__ __forceinline__ float s(int64_t i, int cnt, int k) const { return one(ld1(e, i), ld1(r, i), D.s(i, cnt, k)); }
    __device__ __forceinline__ float4 v(int64_t i, int cnt) const
    {
        const float4 a = ld4(e, i), b = ld4(r, i), d = D.v(i, cnt);
        return make_float4(one(a.x, b.x, d.x), one(a.y, b.y, d.y), one(a.z, b.z, d.z), one(a.w, b.w, d.w));
    }
};
struct SrcScaled {                // sc * p
    const float* p; float sc;
    __device__ __forceinline__ float s(int64_t i, int, int) const { return __fmul_rn(sc, ld1(p, i)); }
    __device__ __forceinline__ float4 v(int64_t i, int) const
    {
        const float4 a = ld4(p, i);
        return make_float4(__fmul_rn(sc, a.x), __fmul_rn(sc, a.y), __fmul_rn(sc, a.z), __fmul_rn(sc, a.w));
    }
};

// x-window of a row: w[0..5] = S(c0-1 .. c0+4), centre values given; periodic wrap in x.
template <class Src>
__device__ __forceinline__ void xwin(const Src& S, const Grid& g, int64_t row, int c0, int cnt, const float (&cen)[4], float (&w)[6])
{
    const int n = g.n[0], per = g.per[0];
    w[1] = cen[0]; w[2] = cen[1]; w[3] = cen[2]; w[4] = cen[3];
    w[0] = S.s(row + ((c0 == 1 && per) ? n : c0 - 1), cnt, 0);
    int ch = c0 + 4;
    if (ch > n + 1) ch = n + 1;                  // beyond the row: value unused
    if (ch == n + 1 && per) ch = 1;
    w[5] = S.s(row + ch, cnt, 5);
    if (per && c0 + 3 > n) {                     // partial last group: cell n+1 lies inside the vector
        float first = S.s(row + 1, cnt, 0);
#pragma unroll
        for (int k = 1; k <= 3; ++k) if (c0 + k == n + 1) w[k + 1] = first;
    }
}

// face coefficients of the thread's four cells on one plane
struct Coef { float x[5], y[4], yp[4], z[4], zp[4]; };

template <int ND, int MODE>
__device__ __forceinline__ void coef_load(const Grid& g, const float* L, float Lc, int64_t i, Coef& C, bool first, const VPos& p, int z)
{
    if (MODE == TM_PLI) {
#pragma unroll
        for (int k = 0; k < 4; ++k) { C.x[k] = Lc; C.y[k] = Lc; C.yp[k] = Lc; C.z[k] = Lc; C.zp[k] = Lc; }
        C.x[4] = Lc;
        return;
    }
    if (MODE == TM_PLB) {
        if (first) {
#pragma unroll
            for (int k = 0; k < 5; ++k) C.x[k] = (!g.per[0] && (p.c0 + k == 1 || p.c0 + k == g.n[0] + 1)) ? 0.0f : Lc;
            const float lo = (!g.per[1] && p.c1 == 1) ? 0.0f : Lc, hi = (!g.per[1] && p.c1 == g.n[1]) ? 0.0f : Lc;
#pragma unroll
            for (int k = 0; k < 4; ++k) { C.y[k] = lo; C.yp[k] = hi; }
        }
        if (ND == 3) {
            const float lo = (!g.per[2] && z == 1) ? 0.0f : Lc, hi = (!g.per[2] && z == g.n[2]) ? 0.0f : Lc;
#pragma unroll
            for (int k = 0; k < 4; ++k) { C.z[k] = lo; C.zp[k] = hi; }
        }
        return;
    }
    float4 a = ld4(L, i);
    C.x[0] = a.x; C.x[1] = a.y; C.x[2] = a.z; C.x[3] = a.w; C.x[4] = ld1(L, i + 4);
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

// Marches one tile: for every plane calls F(z, idx, cnt, w, q[4]) with w = x-window of the operand,
// q = A operand at the thread's four cells and cnt = number of y/z boundary faces of the row.
template <int ND, int MODE, class Src, class Fn>
__device__ __forceinline__ void march(const Grid& g, const VPos& p, const Src& S, const float* L, float Lc, const Ana<ND>& A, Fn&& F)
{
    const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy;
    const int64_t rm = (int64_t)WL_OFF + (int64_t)nb_lo(p.c1, g.n[1], g.per[1]) * g.sy;
    const int64_t rp = (int64_t)WL_OFF + (int64_t)nb_hi(p.c1, g.n[1], g.per[1]) * g.sy;
    float zm[4] = { 0.f, 0.f, 0.f, 0.f }, zc[4], zp[4] = { 0.f, 0.f, 0.f, 0.f };
    int bzm = 0, bzc = 0, bzp = 0;           // boundary-face counts of planes z-1, z, z+1 (TM_PLB only)
    if (MODE == TM_PLB) { bzm = A.bz(g, p.z0 - 1); bzc = A.bz(g, p.z0); }
    if (ND == 3) unpack4(S.v(rc + p.c0 + (int64_t)nb_lo(p.z0, g.n[2], g.per[2]) * g.sz, A.by[1] + bzm), zm);
    unpack4(S.v(rc + p.c0 + (int64_t)p.z0 * g.sz, A.by[1] + bzc), zc);
    Coef C;
    for (int z = p.z0; z <= p.z1; ++z) {
        const int64_t zo = (int64_t)z * g.sz;
        if (MODE == TM_PLB) bzp = A.bz(g, z + 1);
        float w[6], ym[4], yp[4];
        xwin(S, g, rc + zo, p.c0, A.by[1] + bzc, zc, w);
        unpack4(S.v(rm + zo + p.c0, A.by[0] + bzc), ym);
        unpack4(S.v(rp + zo + p.c0, A.by[2] + bzc), yp);
        if (ND == 3) unpack4(S.v(rc + p.c0 + (int64_t)nb_hi(z, g.n[2], g.per[2]) * g.sz, A.by[1] + bzp), zp);
        coef_load<ND, MODE>(g, L, Lc, rc + zo + p.c0, C, z == p.z0, p, z);
        float q[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) q[k] = stencil<ND>(C, k, w, ym, yp, zm, zp);
        F(z, rc + zo + p.c0, A.by[1] + bzc, w, q);
        if (ND == 3) {
#pragma unroll
            for (int k = 0; k < 4; ++k) { zm[k] = zc[k]; zc[k] = zp[k]; }
            bzm = bzc; bzc = bzp;
        }
    }
}

// runs fn<MODE>() for the tile's mode
#define TILE_MODES(mode, CALL)                     \
    do {                                           \
        if ((mode) == TM_PLI) { CALL(TM_PLI); }    \
        else if ((mode) == TM_PLB) { CALL(TM_PLB); } \
        else { CALL(TM_GEN); }                     \
    } while (0)

// ---------------------------------------------------------------- diagonal + uniform flags
// D = -sum_i (L[c,i] + L[c+d_i,i]); iD = 1/D if |D| > 2n*1e-6 else 0 (R-O).  A tile is uniform
// when every face coefficient of every cell in it has its body-free value.  flags[tile]: bit 0 = uniform; bits 1..6 = the
// layer of cells along the tile's -x, +x, -y, +y, -z, +z face holds a cell that is not (what the tile beyond that face has to
// know, k_plain_mode).
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_diag_flags(Grid g, VT vt, const float* __restrict__ L, float Lc, float* __restrict__ iD, int* __restrict__ uniform,
                                                      int* __restrict__ tile_live, CellBox B, PcgScal* sc, RedBuf rb)
{
    __shared__ int live_s, bad_s;
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        {   // a tile no cell of which lies in the box where L may have changed keeps its 1/D, its flag and its count
            const int lx4 = 4 << vt.lxl, ly = WL_VB >> vt.lxl;
            const int tix = tile % vt.ntx, tiy = (tile / vt.ntx) % vt.nty;
            const bool in = 1 + lx4 * tix <= B.hi[0] && lx4 * (tix + 1) >= B.lo[0] && 1 + ly * tiy <= B.hi[1] && ly * (tiy + 1) >= B.lo[1]
                            && p.z0 <= B.hi[2] && p.z1 >= B.lo[2];
            if (!in) {
                if (threadIdx.x == 0) v[0] += (double)tile_live[tile];
                continue;
            }
        }
        if (threadIdx.x == 0) { live_s = 0; bad_s = 0; }
        __syncthreads();
        int bad = 0, cnt = 0;
        if (p.nv > 0) {
            const int lx4 = 4 << vt.lxl, ly = WL_VB >> vt.lxl;
            const int xlo = 1 + lx4 * (tile % vt.ntx), xhi = min(xlo + lx4 - 1, g.n[0]);
            const int ylo = 1 + ly * ((tile / vt.ntx) % vt.nty), yhi = min(ylo + ly - 1, g.n[1]);
            const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy;
            Coef C, R;
            for (int z = p.z0; z <= p.z1; ++z) {
                const int64_t i = rc + (int64_t)z * g.sz + p.c0;
                coef_load<ND, TM_GEN>(g, L, Lc, i, C, z == p.z0, p, z);
                coef_load<ND, TM_PLB>(g, L, Lc, i, R, z == p.z0, p, z);
                float d[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    float D = 0.0f;
                    D -= C.x[k] + C.x[k + 1];
                    D -= C.y[k] + C.yp[k];
                    if (ND == 3) D -= C.z[k] + C.zp[k];
                    d[k] = fabsf(D) > 2.0f * ND * 1e-6f ? 1.0f / D : 0.0f;
                    if (k < p.nv && d[k] != 0.0f) ++cnt;
                    if (k < p.nv) {
                        bool same = C.x[k] == R.x[k] && C.x[k + 1] == R.x[k + 1] && C.y[k] == R.y[k] && C.yp[k] == R.yp[k];
                        if (ND == 3) same = same && C.z[k] == R.z[k] && C.zp[k] == R.zp[k];
                        if (!same) {
                            bad |= 1;
                            if (p.c0 + k == xlo) bad |= 2;
                            if (p.c0 + k == xhi) bad |= 4;
                            if (p.c1 == ylo) bad |= 8;
                            if (p.c1 == yhi) bad |= 16;
                            if (ND == 3 && z == p.z0) bad |= 32;
                            if (ND == 3 && z == p.z1) bad |= 64;
                        }
                    }
                }
                st4(iD, i, d, p.nv);
            }
        }
        v[0] += (double)cnt;
        if (cnt) atomicAdd(&live_s, cnt);
        if (bad) atomicOr(&bad_s, bad);
        __syncthreads();
        if (threadIdx.x == 0) { uniform[tile] = bad_s ^ 1; tile_live[tile] = live_s; }
        __syncthreads();
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) sc->nlive = v[0];
    }
}

// The PCG passes recompute e' = beta e + iD r at the six neighbours of every cell, so a tile may
// only use analytic coefficients if the cells one step outside it are body-free too: its mode is
// TM_GEN unless it is uniform and so is the layer of cells that each face-neighbour tile (periodic wrap) turns
// towards it.  A missing neighbour is a non-periodic domain boundary, whose faces carry L = 0 (R-O) and need no
// values beyond.
__global__ void k_plain_mode(Grid g, VT vt, const int* __restrict__ self, int* __restrict__ plain)
{
    for (int tile = blockIdx.x * blockDim.x + threadIdx.x; tile < vt.ntiles; tile += gridDim.x * blockDim.x) {
        int t[3] = { tile % vt.ntx, (tile / vt.ntx) % vt.nty, tile / (vt.ntx * vt.nty) };
        const int nt[3] = { vt.ntx, vt.nty, vt.ntz };
        int ok = self[tile] & 1;
        for (int d = 0; d < 3 && ok; ++d)
            for (int s = -1; s <= 1; s += 2) {
                int q[3] = { t[0], t[1], t[2] };
                q[d] += s;
                if (q[d] < 0 || q[d] >= nt[d]) {
                    if (!g.per[d]) continue;
                    q[d] = q[d] < 0 ? nt[d] - 1 : 0;
                }
                // the neighbour beyond my +d face shows me its -d layer (bit 1 + 2d), the one beyond my -d face its +d layer
                ok = ok && !((self[q[0] + vt.ntx * (q[1] + vt.nty * q[2])] >> (s > 0 ? 1 + 2 * d : 2 + 2 * d)) & 1);
            }
        int mode = TM_GEN;
        if (ok) {
            // cell range of the tile, one cell wider: does it reach a non-periodic boundary cell?
            const int nd = g.sz == 0 ? 2 : 3;
            const int ext[3] = { 4 << vt.lxl, WL_VB >> vt.lxl, vt.zc };
            mode = TM_PLI;
            for (int d = 0; d < nd; ++d) {
                if (g.per[d]) continue;
                const int lo = 1 + t[d] * ext[d], hi = lo + ext[d] - 1;
                if (lo - 1 <= 1 || hi + 1 >= g.n[d]) mode = TM_PLB;
            }
        }
        plain[tile] = mode;
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

// sum of the thread's (valid) values of r over the coupled cells (iD != 0); uniform tiles have no others
template <int MODE>
__device__ __forceinline__ float live_sum(const float* iD, int64_t i, const float (&ro)[4], int nv)
{
    float d[4] = { 1.f, 1.f, 1.f, 1.f };
    if (MODE == TM_GEN) unpack4(ld4(iD, i), d);
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) if (k < nv && d[k] != 0.0f) s += ro[k];
    return s;
}

// ---------------------------------------------------------------- project!, first half
// (R-K): pscale = w dt; x = pscale p; r = div u - A x.
template <int ND, int MODE>
__device__ __forceinline__ void residual_tile(const Grid& g, const VPos& p, const float* u, const float* L, float Lc, const float* iD,
                                              const float* pr, float sc, float* x, float* r, double& rsum)
{
    SrcScaled S{ pr, sc };
    Ana<ND> A;
    A.init(g, Lc, p);
    float uzc[4] = { 0.f, 0.f, 0.f, 0.f };
    if (ND == 3) unpack4(ld4(u + 2 * g.nalloc, (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + (int64_t)p.z0 * g.sz + p.c0), uzc);
    march<ND, MODE>(g, p, S, L, Lc, A, [&](int z, int64_t i, int, const float (&w)[6], const float (&q)[4]) {
        // u ghosts are BC-filled: plain +1 neighbours
        float ux[4], uy[4], uyp[4], uzp[4] = { 0.f, 0.f, 0.f, 0.f }, xo[4], ro[4];
        unpack4(ld4(u, i), ux);
        const float ux4 = ld1(u, i + 4);
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
        rsum += (double)live_sum<MODE>(iD, i, ro, p.nv);
    });
}

template <int ND>
__global__ void __launch_bounds__(WL_VB, WL_R_MINB) k_residual(Grid g, VT vt, const int* __restrict__ plain, const float* __restrict__ u, const float* __restrict__ L, float Lc,
                                                    const float* __restrict__ iD, const float* __restrict__ p, float* __restrict__ x, float* __restrict__ r,
                                                    DevScal* ds, float w, RedBuf rb)
{
    const float sc = w * ds->dt;
    if (blockIdx.x == 0 && threadIdx.x == 0) ds->pscale = sc;
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos ps = vt_pos(g, vt, tile);
        if (ps.nv == 0) continue;
#define CALL(M) residual_tile<ND, M>(g, ps, u, L, Lc, iD, p, sc, x, r, v[0])
        TILE_MODES(plain[tile], CALL);
#undef CALL
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) ds->pcg[0].rsum = v[0];
    }
}

// ---------------------------------------------------------------- project!, second half
// (P:88 kernel): u[c,i] -= L[c,i] (x[c] - x[c-d_i]); p = x / pscale
// PEND: the smoother left its last update to this kernel (wl_pcgfused.cu): x stands for x + a e wherever it is read (x itself is not
// rewritten: the next solve starts from p).
template <int ND, int MODE, int PEND>
__device__ __forceinline__ void gradient_tile(const Grid& g, const VPos& p, float* u, const float* L, float Lc,
                                              const float* xa, float* pr, float isc, const float* e, float a)
{
    struct {
        const float* x; const float* e; float a;
        __device__ __forceinline__ float4 v(int64_t j) const
        {
            float4 t = ld4(x, j);
            if (PEND) { const float4 s = ld4(e, j); t.x = t.x + a * s.x; t.y = t.y + a * s.y; t.z = t.z + a * s.z; t.w = t.w + a * s.w; }
            return t;
        }
        __device__ __forceinline__ float s(int64_t j) const { float t = ld1(x, j); if (PEND) t = t + a * ld1(e, j); return t; }
    } X = { xa, e, a };
    const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy;
    const int64_t rm = (int64_t)WL_OFF + (int64_t)nb_lo(p.c1, g.n[1], g.per[1]) * g.sy;
    float zm[4] = { 0.f, 0.f, 0.f, 0.f };
    if (ND == 3) unpack4(X.v(rc + p.c0 + (int64_t)nb_lo(p.z0, g.n[2], g.per[2]) * g.sz), zm);
    Coef C;
    for (int z = p.z0; z <= p.z1; ++z) {
        const int64_t i = rc + (int64_t)z * g.sz + p.c0;
        float xc[4], ym[4], o[4];
        unpack4(X.v(i), xc);
        const float xm = X.s(rc + (int64_t)z * g.sz + ((p.c0 == 1 && g.per[0]) ? g.n[0] : p.c0 - 1));
        unpack4(X.v(rm + (int64_t)z * g.sz + p.c0), ym);
        float l[4] = { Lc, Lc, Lc, Lc }, uu[4];
        if (MODE == TM_PLB) coef_load<ND, TM_PLB>(g, L, Lc, i, C, z == p.z0, p, z);
        // x component
        if (MODE == TM_GEN) unpack4(ld4(L, i), l);
        if (MODE == TM_PLB) { l[0] = C.x[0]; l[1] = C.x[1]; l[2] = C.x[2]; l[3] = C.x[3]; }
        unpack4(*reinterpret_cast<const float4*>(u + i), uu);
#pragma unroll
        for (int k = 0; k < 4; ++k) o[k] = uu[k] - l[k] * (xc[k] - (k == 0 ? xm : xc[k - 1]));
        st4(u, i, o, p.nv);
        // y component
        if (MODE == TM_GEN) unpack4(ld4(L + g.nalloc, i), l);
        if (MODE == TM_PLB) { l[0] = C.y[0]; l[1] = C.y[1]; l[2] = C.y[2]; l[3] = C.y[3]; }
        unpack4(*reinterpret_cast<const float4*>(u + g.nalloc + i), uu);
#pragma unroll
        for (int k = 0; k < 4; ++k) o[k] = uu[k] - l[k] * (xc[k] - ym[k]);
        st4(u + g.nalloc, i, o, p.nv);
        if (ND == 3) {
            if (MODE == TM_GEN) unpack4(ld4(L + 2 * g.nalloc, i), l);
            if (MODE == TM_PLB) { l[0] = C.z[0]; l[1] = C.z[1]; l[2] = C.z[2]; l[3] = C.z[3]; }
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
__global__ void __launch_bounds__(WL_VB, WL_G_MINB) k_apply_gradient(Grid g, VT vt, const int* __restrict__ plain, float* __restrict__ u, const float* __restrict__ L, float Lc,
                                                          const float* __restrict__ x, float* __restrict__ p, const DevScal* __restrict__ ds)
{
    const float isc = 1.0f / ds->pscale;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos ps = vt_pos(g, vt, tile);
        if (ps.nv == 0) continue;
#define CALL(M) gradient_tile<ND, M, 0>(g, ps, u, L, Lc, x, p, isc, nullptr, 0.0f)
        TILE_MODES(plain[tile], CALL);
#undef CALL
    }
}

// the same with the smoother's last update x += alpha e (iteration kprev) applied on the fly; the update is owed under the
// conditions of k_pcg_last: the smoother is live, or it stopped in that very iteration
template <int ND>
__global__ void __launch_bounds__(WL_VB, WL_G_MINB) k_apply_gradient_pend(Grid g, VT vt, const int* __restrict__ plain, float* __restrict__ u, const float* __restrict__ L, float Lc,
                                                               const float* __restrict__ x, float* __restrict__ p, const DevScal* __restrict__ ds,
                                                               const float* __restrict__ e, const PcgScal* __restrict__ sc, int kprev)
{
    const float isc = 1.0f / ds->pscale;
    const bool owed = sc->live || sc->stop_k == kprev;
    const float a = (float)sc->alpha;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos ps = vt_pos(g, vt, tile);
        if (ps.nv == 0) continue;
        if (owed) {
#define CALL(M) gradient_tile<ND, M, 1>(g, ps, u, L, Lc, x, p, isc, e, a)
            TILE_MODES(plain[tile], CALL);
#undef CALL
        } else {
#define CALL(M) gradient_tile<ND, M, 0>(g, ps, u, L, Lc, x, p, isc, nullptr, 0.0f)
            TILE_MODES(plain[tile], CALL);
#undef CALL
        }
    }
}

// ---------------------------------------------------------------- residual restriction
// r_c[C] = sum of the 2^n children; x_c = 0 (R-S).  One thread per four coarse cells.
// PEND: the fine level's smoother left its last update to its readers (wl_pcgfused.cu): r stands for r - a q
template <int ND, int MODE, int PEND = 0>
__device__ __forceinline__ void restrict_tile(const Grid& gf, const Grid& gc, const VPos& p, const float* rf, const float* iDc_arr, float* rc, float* xc, double& rsum,
                                              const float* qf = nullptr, float a = 0.0f)
{
    const int f0 = 2 * p.c0 - 1, f1 = 2 * p.c1 - 1;      // first fine child (f0 = 1 + 8 gx: 32-byte aligned)
    for (int z = p.z0; z <= p.z1; ++z) {
        float s[4] = { 0.f, 0.f, 0.f, 0.f };
        const int nz = ND == 3 ? 2 : 1;
        for (int a2 = 0; a2 < nz; ++a2)
            for (int a1 = 0; a1 < 2; ++a1) {
                const int64_t b = gidx(gf, f0, f1 + a1, ND == 3 ? 2 * z - 1 + a2 : 0);
                float4 lo = ld4(rf, b);
                if (PEND) { const float4 t = ld4(qf, b); lo.x = __fmaf_rn(-a, t.x, lo.x); lo.y = __fmaf_rn(-a, t.y, lo.y); lo.z = __fmaf_rn(-a, t.z, lo.z); lo.w = __fmaf_rn(-a, t.w, lo.w); }
                s[0] += lo.x; s[0] += lo.y; s[1] += lo.z; s[1] += lo.w;
                if (p.nv > 2) {
                    float4 hi = ld4(rf, b + 4);
                    if (PEND) { const float4 t = ld4(qf, b + 4); hi.x = __fmaf_rn(-a, t.x, hi.x); hi.y = __fmaf_rn(-a, t.y, hi.y); hi.z = __fmaf_rn(-a, t.z, hi.z); hi.w = __fmaf_rn(-a, t.w, hi.w); }
                    s[2] += hi.x; s[2] += hi.y; s[3] += hi.z; s[3] += hi.w;
                }
            }
        const int64_t i = gidx(gc, p.c0, p.c1, z);
        const float zero[4] = { 0.f, 0.f, 0.f, 0.f };
        st4(rc, i, s, p.nv);
        st4(xc, i, zero, p.nv);
        rsum += (double)live_sum<MODE>(iDc_arr, i, s, p.nv);
    }
}

// vt, plain, iD belong to the COARSE level
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_restrict_r(Grid gf, Grid gc, VT vt, const int* __restrict__ plain, const float* __restrict__ rf, const float* __restrict__ iD,
                                                      float* __restrict__ rc, float* __restrict__ xc, PcgScal* scc, RedBuf rb)
{
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(gc, vt, tile);
        if (p.nv == 0) continue;
        if (plain[tile] == TM_GEN) restrict_tile<ND, TM_GEN>(gf, gc, p, rf, iD, rc, xc, v[0]);
        else                       restrict_tile<ND, TM_PLI>(gf, gc, p, rf, iD, rc, xc, v[0]);
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) scc->rsum = v[0];
    }
}

// the same with the fine level's pending update (iteration kprev of its smoother; owed as in k_pcg_last)
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_restrict_r_pend(Grid gf, Grid gc, VT vt, const int* __restrict__ plain, const float* __restrict__ rf, const float* __restrict__ iD,
                                                           float* __restrict__ rc, float* __restrict__ xc, PcgScal* scc, RedBuf rb,
                                                           const float* __restrict__ qf, const PcgScal* __restrict__ scf, int kprev)
{
    double v[1] = { 0.0 };
    const bool owed = scf->live || scf->stop_k == kprev;
    const float a = (float)scf->alpha;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(gc, vt, tile);
        if (p.nv == 0) continue;
        const bool gen = plain[tile] == TM_GEN;
        if (owed) {
            if (gen) restrict_tile<ND, TM_GEN, 1>(gf, gc, p, rf, iD, rc, xc, v[0], qf, a);
            else     restrict_tile<ND, TM_PLI, 1>(gf, gc, p, rf, iD, rc, xc, v[0], qf, a);
        } else {
            if (gen) restrict_tile<ND, TM_GEN>(gf, gc, p, rf, iD, rc, xc, v[0]);
            else     restrict_tile<ND, TM_PLI>(gf, gc, p, rf, iD, rc, xc, v[0]);
        }
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) scc->rsum = v[0];
    }
}

// ---------------------------------------------------------------- prolongation + increment
// e = P x_c (piecewise constant); x_f += e; r_f -= A_f e (R-S)
__device__ __forceinline__ int par(int c) { return (c + 1) >> 1; }          // parent of a fine index (ghost 0 -> 0, n+1 -> n/2+1)
__device__ __forceinline__ int wrapC(int C, int n, int per) { if (per) { if (C < 1) C += n; else if (C > n) C -= n; } return C; }

// PEND: x_f stands for x_f + a e and r_f for rin - a q (the fine smoother's last update, left to its readers); the results go to
// xf and rf as always
template <int ND, int MODE, int PEND = 0>
__device__ __forceinline__ void prolong_tile(const Grid& gf, const Grid& gc, const VPos& p, const float* L, float Lc, const float* iD,
                                             const float* xc, float* xf, float* rf, double& rsum,
                                             const float* rin = nullptr, const float* e = nullptr, const float* q = nullptr, float a = 0.0f)
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
        const float v0 = ld1(xc, row + X0), v1 = ld1(xc, row + X1), v2 = ld1(xc, row + X2), v3 = ld1(xc, row + X3);
        const float w[6] = { v0, v1, v1, v2, v2, v3 };
        float ym[4], yp[4], zm[4] = { 0.f, 0.f, 0.f, 0.f }, zp[4] = { 0.f, 0.f, 0.f, 0.f };
        {
            const int64_t a = gidx(gc, 0, Ym, Z), b = gidx(gc, 0, Yp, Z);
            float a1 = ld1(xc, a + X1), a2 = ld1(xc, a + X2), b1 = ld1(xc, b + X1), b2 = ld1(xc, b + X2);
            ym[0] = a1; ym[1] = a1; ym[2] = a2; ym[3] = a2;
            yp[0] = b1; yp[1] = b1; yp[2] = b2; yp[3] = b2;
        }
        if (ND == 3) {
            const int64_t a = gidx(gc, 0, Y, par(nb_lo(z, gf.n[2], gf.per[2]))), b = gidx(gc, 0, Y, par(nb_hi(z, gf.n[2], gf.per[2])));
            float a1 = ld1(xc, a + X1), a2 = ld1(xc, a + X2), b1 = ld1(xc, b + X1), b2 = ld1(xc, b + X2);
            zm[0] = a1; zm[1] = a1; zm[2] = a2; zm[3] = a2;
            zp[0] = b1; zp[1] = b1; zp[2] = b2; zp[3] = b2;
        }
        coef_load<ND, MODE>(gf, L, Lc, i, C, z == p.z0, p, z);
        float xo[4], ro[4];
        unpack4(*reinterpret_cast<const float4*>(xf + i), xo);
        if (PEND == 1) {
            float ee[4], qq[4];
            unpack4(*reinterpret_cast<const float4*>(rin + i), ro);
            unpack4(ld4(e, i), ee); unpack4(ld4(q, i), qq);
#pragma unroll
            for (int k = 0; k < 4; ++k) { xo[k] += a * ee[k]; ro[k] = __fmaf_rn(-a, qq[k], ro[k]); }
        } else if (PEND == 2) unpack4(*reinterpret_cast<const float4*>(rin + i), ro);      // nothing owed: r only changes buffers
        else unpack4(*reinterpret_cast<const float4*>(rf + i), ro);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            xo[k] += w[k + 1];
            ro[k] -= stencil<ND>(C, k, w, ym, yp, zm, zp);
        }
        st4(xf, i, xo, p.nv);
        st4(rf, i, ro, p.nv);
        rsum += (double)live_sum<MODE>(iD, i, ro, p.nv);
    }
}

template <int ND>
__global__ void __launch_bounds__(WL_VB, WL_P_MINB) k_prolong(Grid gf, Grid gc, VT vt, const int* __restrict__ plain, const float* __restrict__ L, float Lc, const float* __restrict__ iD,
                                                   const float* __restrict__ xc, float* __restrict__ xf, float* __restrict__ rf, PcgScal* scf, RedBuf rb)
{
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(gf, vt, tile);
        if (p.nv == 0) continue;
#define CALL(M) prolong_tile<ND, M>(gf, gc, p, L, Lc, iD, xc, xf, rf, v[0])
        TILE_MODES(plain[tile], CALL);
#undef CALL
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) scf->rsum = v[0];
    }
}

template <int ND>
__global__ void __launch_bounds__(WL_VB, WL_P_MINB) k_prolong_pend(Grid gf, Grid gc, VT vt, const int* __restrict__ plain, const float* __restrict__ L, float Lc, const float* __restrict__ iD,
                                                        const float* __restrict__ xc, float* __restrict__ xf, float* __restrict__ rf, PcgScal* scf, RedBuf rb,
                                                        const float* rin, const float* __restrict__ e, const float* __restrict__ q, int kprev)
{
    double v[1] = { 0.0 };
    const bool owed = scf->live || scf->stop_k == kprev;
    const float a = owed ? (float)scf->alpha : 0.0f;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(gf, vt, tile);
        if (p.nv == 0) continue;
        if (owed) {
#define CALL(M) prolong_tile<ND, M, 1>(gf, gc, p, L, Lc, iD, xc, xf, rf, v[0], rin, e, q, a)
            TILE_MODES(plain[tile], CALL);
#undef CALL
        } else if (rin != rf) {       // nothing owed, but the residual sits in the other buffer
#define CALL(M) prolong_tile<ND, M, 2>(gf, gc, p, L, Lc, iD, xc, xf, rf, v[0], rin, e, q, a)
            TILE_MODES(plain[tile], CALL);
#undef CALL
        } else {
#define CALL(M) prolong_tile<ND, M>(gf, gc, p, L, Lc, iD, xc, xf, rf, v[0])
            TILE_MODES(plain[tile], CALL);
#undef CALL
        }
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) scf->rsum = v[0];
    }
}

// ---------------------------------------------------------------- Jacobi-PCG smoother
// (R-S, R-T), restarted at every call:
//   z = e = iD r; rho = r.z; if |rho| < tau return
//   loop k = 1..it: q = A e; gamma = q.e; alpha = rho/gamma; x += alpha e; r -= alpha q;
//                   if k == it break; z = iD r; rho' = r.z; if |rho'| < tau or < theta |rho0| break;
//                   beta = rho'/rho; e = beta e + z; rho = rho'
// Dot products: fp32 products summed over the thread's four cells, then accumulated in fp64.
__device__ __forceinline__ float pcg_mean(const PcgScal* sc) { return sc->nlive > 0.0 ? (float)(sc->rsum / sc->nlive) : 0.0f; }

template <int ND, int FIRST, int MODE>
__device__ __forceinline__ void pcgA_tile(const Grid& g, const VPos& p, const float* L, float Lc, float iDc,
                                          const float* ein, const float* r, const float* iD, float beta, float m,
                                          float* eout, float* q, double& gam, double& rho)
{
    Ana<ND> A;
    A.init(g, Lc, p);
    auto body = [&](int z, int64_t i, int, const float (&w)[6], const float (&qq)[4]) {
        float eo[4] = { w[1], w[2], w[3], w[4] };
        st4(eout, i, eo, p.nv);
        st4(q, i, qq, p.nv);
        float rr[4] = { 0.f, 0.f, 0.f, 0.f };
        if (FIRST) unpack4(ld4(r, i), rr);
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (k < p.nv) {
                gam += (double)qq[k] * (double)eo[k];
                if (FIRST) rho += (double)eo[k] * (double)(rr[k] - m);
            }
    };
    IDiag<ND, MODE> D{ iD, iDc, &A };
    if (FIRST) { SrcFirst<ND, MODE> S{ r, D, m }; march<ND, MODE>(g, p, S, L, Lc, A, body); }
    else       { SrcNext<ND, MODE> S{ ein, r, D, beta }; march<ND, MODE>(g, p, S, L, Lc, A, body); }
}

// x += alpha e; r = (r - m) - alpha q on the coupled cells (m = 0 after the first iteration); unless last: rho' += r.(iD r)
template <int ND, int MODE>
__device__ __forceinline__ void pcgB_tile(const Grid& g, const VPos& p, float Lc, float iDc, float alpha, float m, float* x, float* r,
                                          const float* e, const float* q, const float* iD, int last, double& rho2)
{
    Ana<ND> A;
    A.init(g, Lc, p);
    IDiag<ND, MODE> D{ iD, iDc, &A };
    const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + p.c0;
    for (int z = p.z0; z <= p.z1; ++z) {
        const int64_t i = rc + (int64_t)z * g.sz;
        float xo[4], ro[4], ee[4], qq[4], dd[4] = { 0.f, 0.f, 0.f, 0.f };
        unpack4(*reinterpret_cast<const float4*>(x + i), xo);
        unpack4(*reinterpret_cast<const float4*>(r + i), ro);
        unpack4(ld4(e, i), ee);
        unpack4(ld4(q, i), qq);
        if (!last || m != 0.0f) unpack4(D.v(i, A.by[1] + A.bz(g, z)), dd);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            xo[k] += alpha * ee[k];
            if (m != 0.0f && dd[k] != 0.0f) ro[k] -= m;
            ro[k] -= alpha * qq[k];
            if (!last && k < p.nv) rho2 += (double)__fmul_rn(dd[k], ro[k]) * (double)ro[k];
        }
        st4(x, i, xo, p.nv);
        st4(r, i, ro, p.nv);
    }
}

template <int ND, int FIRST>
__global__ void __launch_bounds__(WL_VB, WL_A_MINB) k_pcg_A(Grid g, VT vt, const int* __restrict__ plain, const float* __restrict__ L, float Lc, float iDc,
                                                 const float* __restrict__ ein, const float* __restrict__ r, const float* __restrict__ iD,
                                                 float* __restrict__ eout, float* __restrict__ q, PcgScal* sc, RedBuf rb)
{
    if (!FIRST && !sc->live) return;          // uniform across the grid: written by an earlier kernel
    const float beta = FIRST ? 0.0f : (float)sc->beta;
    const float m = FIRST ? pcg_mean(sc) : 0.0f;
    double v[2] = { 0.0, 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
#define CALL(M) pcgA_tile<ND, FIRST, M>(g, p, L, Lc, iDc, ein, r, iD, beta, m, eout, q, v[0], v[1])
        TILE_MODES(plain[tile], CALL);
#undef CALL
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

template <int ND>
__global__ void __launch_bounds__(WL_VB, WL_B_MINB) k_pcg_B(Grid g, VT vt, const int* __restrict__ plain, float Lc, float iDc, float* __restrict__ x, float* __restrict__ r,
                                                 const float* __restrict__ e, const float* __restrict__ q, const float* __restrict__ iD,
                                                 PcgScal* sc, RedBuf rb, int first, int last)
{
    if (!sc->live) return;
    const float alpha = (float)sc->alpha;
    const float m = first ? pcg_mean(sc) : 0.0f;
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
#define CALL(M) pcgB_tile<ND, M>(g, p, Lc, iDc, alpha, m, x, r, e, q, iD, last, v[0])
        TILE_MODES(plain[tile], CALL);
#undef CALL
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

// sum of r over the coupled cells of a level (stage hooks only: in a solve the kernel that writes r leaves it)
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_rsum(Grid g, VT vt, const int* __restrict__ plain, const float* __restrict__ r, const float* __restrict__ iD, PcgScal* sc, RedBuf rb)
{
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
        const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + p.c0;
        for (int z = p.z0; z <= p.z1; ++z) {
            const int64_t i = rc + (int64_t)z * g.sz;
            float ro[4];
            unpack4(ld4(r, i), ro);
            v[0] += (double)(plain[tile] == TM_GEN ? live_sum<TM_GEN>(iD, i, ro, p.nv) : live_sum<TM_PLI>(iD, i, ro, p.nv));
        }
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) sc->rsum = v[0];
    }
}

// ================================================================== the coarse levels: one persistent kernel
// Below the fine level(s) a V-cycle is a long chain of short dependent passes (restrict, 2 x 6 PCG
// passes per level, prolong), each far too small to fill the GPU: as separate launches they cost
// launch latency + a grid-wide tail each.  k_coarse runs the whole chain as ONE cooperative launch:
// co-resident blocks walk the tiles of every pass and meet at a grid barrier between passes; the dot
// products are summed from per-block partials in a fixed order by every block (bit-identical in all
// blocks, so every block takes the same branches of the PCG guards).  The passes are the same tile
// functions the fine-level kernels use.
struct PkCtx {
    double* part;        // [2][WL_MAX_PARTIALS][WL_PK_SLOT] per-block partial sums (one slot per block), alternating by reduction
    int phase;
};
#define PK_NV 2

// barrier over all blocks of the cooperative launch: every global write before it is visible to every block after it
// (3.2 us on B200)
__device__ __forceinline__ void pk_barrier(PkCtx&) { cooperative_groups::this_grid().sync(); }

// grid-wide sum of NV values; includes a grid barrier (all writes before it are visible after it)
template <int NV>
__device__ __forceinline__ void pk_reduce(PkCtx& c, double (&v)[NV])
{
    __shared__ double sm[PK_NV][32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = WL_VB >> 5;
    double* part = c.part + (size_t)(c.phase & 1) * WL_PK_SLOT * WL_MAX_PARTIALS;
    c.phase++;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double w = warp_red<OpSum>(v[k]);
        if (lane == 0) sm[k][wid] = w;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double w = lane < nw ? sm[k][lane] : 0.0;
            w = warp_red<OpSum>(w);
            if (lane == 0) part[blockIdx.x * WL_PK_SLOT + k] = w;
        }
    }
    pk_barrier(c);
    // every block adds all partials in the same fixed order: thread-strided (all loads in flight at once; a
    // single warp walking the list pays one L2 round trip per step), then the same warp/shared tree as above
    {
        double w[NV][2];
        const int G = (int)gridDim.x;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int b = tid + j * WL_VB;
#pragma unroll
            for (int k = 0; k < NV; ++k) w[k][j] = b < G ? __ldcg(&part[b * WL_PK_SLOT + k]) : 0.0;
        }
#pragma unroll
        for (int k = 0; k < NV; ++k) {
            double t = w[k][0] + w[k][1];
            for (int b = tid + 2 * WL_VB; b < G; b += WL_VB) t += __ldcg(&part[b * WL_PK_SLOT + k]);   // grids beyond 512 blocks
            t = warp_red<OpSum>(t);
            if (lane == 0) sm[k][wid] = t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < (WL_VB >> 5); ++i) t += sm[k][i];
        v[k] = t;
    }
    __syncthreads();
}

template <int ND>
__device__ __forceinline__ void pk_smooth(PkCtx& c, const LevDev& lv, PcgScal* sc, int iters, double rsum)
{
    const Grid& g = lv.g;
    const VT& vt = lv.vt;
    const double nlive = sc->nlive;
    const float m = nlive > 0.0 ? (float)(rsum / nlive) : 0.0f;
    float* ea = lv.e;
    float* eb = lv.e2;
    double rho = 0.0, rho0 = 0.0, beta = 0.0;
    for (int k = 1; k <= iters; ++k) {
        double v[2] = { 0.0, 0.0 };
        for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
            VPos p = vt_pos(g, vt, tile);
            if (p.nv == 0) continue;
            const int mode = lv.plain[tile];
            if (k == 1) {
#define CALL(M) pcgA_tile<ND, 1, M>(g, p, lv.L, lv.Lc, lv.iDc, eb, lv.r, lv.iD, 0.0f, m, ea, lv.q, v[0], v[1])
                TILE_MODES(mode, CALL);
#undef CALL
            } else {
#define CALL(M) pcgA_tile<ND, 0, M>(g, p, lv.L, lv.Lc, lv.iDc, eb, lv.r, lv.iD, (float)beta, 0.0f, ea, lv.q, v[0], v[1])
                TILE_MODES(mode, CALL);
#undef CALL
            }
        }
        pk_reduce<2>(c, v);
        bool live = true;
        if (k == 1) { rho = rho0 = v[1]; live = !(fabs(rho) < WL_TAU); }
        const double gamma = v[0];
        if (gamma == 0.0 || !isfinite(gamma) || !live) return;     // the barrier of pk_reduce is behind us
        const float alpha = (float)(rho / gamma);
        const int last = k == iters;
        double w[1] = { 0.0 };
        for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
            VPos p = vt_pos(g, vt, tile);
            if (p.nv == 0) continue;
#define CALL(M) pcgB_tile<ND, M>(g, p, lv.Lc, lv.iDc, alpha, k == 1 ? m : 0.0f, lv.x, lv.r, ea, lv.q, lv.iD, last, w[0])
            TILE_MODES(lv.plain[tile], CALL);
#undef CALL
        }
        if (last) { pk_barrier(c); return; }
        pk_reduce<1>(c, w);
        const double rho2 = w[0];
        if (fabs(rho2) < WL_TAU || fabs(rho2) < WL_THETA * fabs(rho0)) return;
        beta = rho2 / rho;
        rho = rho2;
        float* t = ea; ea = eb; eb = t;
    }
}

template <int ND>
__device__ __forceinline__ void coarse_body(const LevDev* levs, const CoarseProg& prog, DevScal* ds, double* part)
{
    __shared__ LevDev la, lb;
    PkCtx c;
    c.part = part; c.phase = 0;
    double rsum = 0.0;
    int rsum_level = -1;
    for (int o = 0; o < prog.n; ++o) {
        const CoarseOp op = prog.op[o];
        __syncthreads();
        if (threadIdx.x == 0) {     // level descriptors of this pass into shared memory (typed copies: no punning)
            la = levs[op.level];
            lb = levs[op.level + (op.kind == COP_SMOOTH ? 0 : 1)];
        }
        __syncthreads();
        if (op.kind == COP_SMOOTH) {
            PcgScal* sc = &ds->pcg[op.level];
            const double rs = rsum_level == op.level ? rsum : sc->rsum;
            pk_smooth<ND>(c, la, sc, op.iters, rs);
            rsum = 0.0; rsum_level = op.level;               // the mean of r has been removed (R-T2)
            if (blockIdx.x == 0 && threadIdx.x == 0) sc->rsum = 0.0;
        } else if (op.kind == COP_RESTRICT) {        // la = fine, lb = coarse
            double v[1] = { 0.0 };
            for (int tile = blockIdx.x; tile < lb.vt.ntiles; tile += gridDim.x) {
                VPos p = vt_pos(lb.g, lb.vt, tile);
                if (p.nv == 0) continue;
                if (lb.plain[tile] == TM_GEN) restrict_tile<ND, TM_GEN>(la.g, lb.g, p, la.r, lb.iD, lb.r, lb.x, v[0]);
                else                          restrict_tile<ND, TM_PLI>(la.g, lb.g, p, la.r, lb.iD, lb.r, lb.x, v[0]);
            }
            pk_reduce<1>(c, v);
            rsum = v[0]; rsum_level = op.level + 1;
            if (blockIdx.x == 0 && threadIdx.x == 0) ds->pcg[op.level + 1].rsum = v[0];
        } else {                                     // COP_PROLONG: la = fine, lb = coarse
            double v[1] = { 0.0 };
            for (int tile = blockIdx.x; tile < la.vt.ntiles; tile += gridDim.x) {
                VPos p = vt_pos(la.g, la.vt, tile);
                if (p.nv == 0) continue;
#define CALL(M) prolong_tile<ND, M>(la.g, lb.g, p, la.L, la.Lc, la.iD, lb.x, la.x, la.r, v[0])
                TILE_MODES(la.plain[tile], CALL);
#undef CALL
            }
            pk_reduce<1>(c, v);
            rsum = v[0]; rsum_level = op.level;
            if (blockIdx.x == 0 && threadIdx.x == 0) ds->pcg[op.level].rsum = v[0];
        }
    }
}

template <int ND>
__global__ void __launch_bounds__(WL_VB, WL_PK_MINB) k_coarse(const LevDev* levs, const __grid_constant__ CoarseProg prog, DevScal* ds, double* part)
{
    coarse_body<ND>(levs, prog, ds, part);
}

// The order in which the one-sweep smoother (wl_pcgfused.cu) hands out the tiles of a level: block b of G takes entries b, b + G, ...
// A TM_GEN tile costs about two uniform ones (L and 1/D are loaded), and with the tiles dealt in index order the blocks that met two
// or three of them finished last (C4: 219 us per sweep against 205 without a body).  So the TM_GEN tiles go first, one per block
// as far as they reach, and the uniform tiles follow in index order (neighbouring blocks keep working on neighbouring memory): the
// deal stays static, so the per-block partial sums and with them the results stay the same from run to run.
__global__ void __launch_bounds__(1024) k_tile_sched(int ntiles, const int* __restrict__ plain, int* __restrict__ sched)
{
    __shared__ int cnt[1024];
    const int tid = threadIdx.x, per = (ntiles + 1023) / 1024;
    const int t0 = tid * per < ntiles ? tid * per : ntiles, t1 = t0 + per < ntiles ? t0 + per : ntiles;
    int c = 0;
    for (int t = t0; t < t1; ++t) c += plain[t] == TM_GEN ? 1 : 0;
    cnt[tid] = c;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {       // inclusive scan
        const int v = tid >= o ? cnt[tid - o] : 0;
        __syncthreads();
        cnt[tid] += v;
        __syncthreads();
    }
    const int ngen = cnt[1023];
    int ig = cnt[tid] - c;                     // TM_GEN tiles before t0
    int ip = ngen + (t0 - ig);                 // uniform tiles before t0 come after all the TM_GEN tiles
    for (int t = t0; t < t1; ++t) {
        const int mode = plain[t];
        if (mode == TM_GEN) sched[ig++] = t | (mode << 24);
        else                sched[ip++] = t | (mode << 24);
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

// After a measure! that rewrote only the box the body can reach (wl_k_measure), L, 1/D and the tile flags change only in
// that box grown by one cell, halved and grown by one cell again from level to level.
void wl_k_poisson_update(wl_sim* s)
{
    CellBox B;
    for (int d = 0; d < 3; ++d) {
        const int n = s->lev[0].g.n[d];
        B.lo[d] = s->mbox_lo[d] - 1 < 1 ? 1 : s->mbox_lo[d] - 1;
        B.hi[d] = s->mbox_hi[d] + 1 > n ? n : s->mbox_hi[d] + 1;
        if (d >= s->nd) { B.lo[d] = 0; B.hi[d] = 0; }
    }
    for (int l = 0; l < s->nlev; ++l) {
        Level& lv = s->lev[l];
        if (l > 0) {
            Level& lf = s->lev[l - 1];
            for (int d = 0; d < s->nd; ++d) {
                const int lo = (B.lo[d] + 1) / 2 - 1, hi = (B.hi[d] + 1) / 2 + 1;
                B.lo[d] = lo < 1 ? 1 : lo;
                B.hi[d] = hi > lv.g.n[d] ? lv.g.n[d] : hi;
            }
            int o[3] = { B.lo[0], B.lo[1], s->nd == 3 ? B.lo[2] : 0 };
            int e[3] = { B.hi[0] - B.lo[0] + 2, B.hi[1] - B.lo[1] + 2, s->nd == 3 ? B.hi[2] - B.lo[2] + 2 : 1 };      // faces lo .. hi + 1
            Tiling T = wl_tiling(s->nd, o, e);
            DISPATCH(s, WLK_POISSON_UPDATE, l > 1, k_restrict_L, T, lf.g, lv.g, T, lf.L, lv.L);
        }
        VDISPATCH(s, WLK_POISSON_UPDATE, l > 0, lv.vt, k_diag_flags<2>, k_diag_flags<3>, lv.g, lv.vt, lv.L, lv.Lc, lv.iD, lv.uniform, lv.tile_live, B, &s->ds->pcg[l], s->rb);
        {
            ProfScope ps_(s, WLK_POISSON_UPDATE, l > 0);
            int nb = (lv.vt.ntiles + 255) / 256;
            k_plain_mode<<<nb < 64 ? nb : 64, 256, 0, s->st>>>(lv.g, lv.vt, lv.uniform, lv.plain);
            if (lv.sched) k_tile_sched<<<1, 1024, 0, s->st>>>(lv.vt.ntiles, lv.plain, lv.sched);
        }
    }
}

void wl_k_residual(wl_sim* s, const float* u, float w)
{
    Level& lv = s->lev[0];
    VDISPATCH(s, WLK_RESIDUAL, 0, lv.vt, k_residual<2>, k_residual<3>, lv.g, lv.vt, lv.plain, u, lv.L, lv.Lc, lv.iD, s->p, lv.x, lv.r, s->ds, w, s->rb);
}

void wl_k_apply_gradient(wl_sim* s, float* u)
{
    Level& lv = s->lev[0];
    if (s->pend_e) {
        const float* e = s->pend_e;
        s->pend_e = nullptr;
        VDISPATCH(s, WLK_GRADIENT, 0, lv.vt, k_apply_gradient_pend<2>, k_apply_gradient_pend<3>, lv.g, lv.vt, lv.plain, u, lv.L, lv.Lc, lv.x, s->p, s->ds,
                  e, &s->ds->pcg[0], s->pend_k);
        return;
    }
    VDISPATCH(s, WLK_GRADIENT, 0, lv.vt, k_apply_gradient<2>, k_apply_gradient<3>, lv.g, lv.vt, lv.plain, u, lv.L, lv.Lc, lv.x, s->p, s->ds);
}

// one k_coarse launch (cooperative, whole GPU)
static void coarse_launch_one(wl_sim* s, const CoarseProg& prog)
{
    if (prog.n <= 0) return;
    if (!s->pk_blocks) {
        int per_sm = 0;
        if (s->nd == 3) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_coarse<3>, WL_VB, 0);
        else            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_coarse<2>, WL_VB, 0);
        if (per_sm > WL_PK_MINB) per_sm = WL_PK_MINB;
        if (s->cfg.tune.pk_blocks_per_sm > 0 && s->cfg.tune.pk_blocks_per_sm < per_sm) per_sm = s->cfg.tune.pk_blocks_per_sm;
        if (per_sm < 1) per_sm = 1;
        int nb = per_sm * s->sm_count;
        if (nb > WL_MAX_PARTIALS) nb = WL_MAX_PARTIALS;
        s->pk_blocks = nb;
    }
    ProfScope ps_(s, WLK_COARSE, 1);
    const LevDev* levs = s->levdev;
    DevScal* ds = s->ds;
    double* part = s->pk_part;
    void* args[] = { (void*)&levs, (void*)&prog, (void*)&ds, (void*)&part };
    cudaError_t e = cudaErrorCooperativeLaunchTooLarge;
    if (s->cfg.tune.pk_fail) { }                  // test hook: the device "refuses" the launch
    else if (s->nd == 3) e = cudaLaunchCooperativeKernel((const void*)k_coarse<3>, dim3(s->pk_blocks), dim3(WL_VB), args, 0, s->st);
    else                 e = cudaLaunchCooperativeKernel((const void*)k_coarse<2>, dim3(s->pk_blocks), dim3(WL_VB), args, 0, s->st);
    if (e != cudaSuccess) {
        // the grid cannot be co-scheduled on this device (a partitioned GPU: MIG, an MPS SM limit): from now on every level runs its
        // passes as stand-alone kernels, starting with this chain
        cudaGetLastError();
        s->pk_level = s->nlev;
        s->tiny_on = 0;
        for (int o = 0; o < prog.n; ++o) {
            const CoarseOp& op = prog.op[o];
            if (op.kind == COP_RESTRICT) wl_k_restrict(s, op.level);
            else if (op.kind == COP_PROLONG) wl_k_prolong(s, op.level);
            else { wl_k_rsum(s, op.level); wl_k_smooth(s, op.level, op.iters, 1); }
        }
    }
}

// blocks of the k_small cluster a pass needs (the level whose cells it walks), or 0 when the pass belongs to k_coarse
static int op_small_blocks(wl_sim* s, const CoarseOp& op)
{
    if (!s->tiny_on) return 0;
    if (s->small_cmax < 0) s->small_cmax = wl_small_max_cluster(s);      // once per handle
    const int walked = op.kind == COP_RESTRICT ? op.level + 1 : op.level;
    return wl_small_blocks(s->lev[walked].g, s->small_cmax);
}

// runs a chain of coarse-level passes: consecutive passes of the same kind (whole-GPU cooperative kernel / one on-chip cluster)
// share a launch
static void coarse_launch(wl_sim* s, const CoarseProg& prog)
{
    int i = 0;
    while (i < prog.n) {
        const int small = op_small_blocks(s, prog.op[i]) > 0;
        CoarseProg P; P.n = 0;
        int C = 1;
        while (i < prog.n && (op_small_blocks(s, prog.op[i]) > 0) == small) {
            const int c = op_small_blocks(s, prog.op[i]);
            if (c > C) C = c;
            P.op[P.n++] = prog.op[i++];
        }
        if (small) {
            if (s->cfg.tune.pk_fail || !wl_k_small_prog(s, P, C)) {        // the cluster could not be launched after all: the cooperative kernel from now on
                cudaGetLastError();
                s->small_cmax = 0;
                coarse_launch_one(s, P);
            }
        } else coarse_launch_one(s, P);
    }
}

void wl_k_coarse_prog(wl_sim* s, const CoarseProg& P) { coarse_launch(s, P); }

static void prog_add(CoarseProg& P, int kind, int level, int iters) { P.op[P.n].kind = kind; P.op[P.n].level = level; P.op[P.n].iters = iters; P.n++; }

void wl_k_restrict(wl_sim* s, int l)
{
    Level &lf = s->lev[l], &lc = s->lev[l + 1];
    if (l >= s->pk_level) { CoarseProg P; P.n = 0; prog_add(P, COP_RESTRICT, l, 0); coarse_launch(s, P); return; }
    if (l == 0 && s->pr_r) {       // the smoother's last update is still pending (wl_pcgfused.cu): r = pr_r - alpha pr_q
        VDISPATCH(s, WLK_RESTRICT, 0, lc.vt, k_restrict_r_pend<2>, k_restrict_r_pend<3>, lf.g, lc.g, lc.vt, lc.plain, s->pr_r, lc.iD, lc.r, lc.x, &s->ds->pcg[1], s->rb,
                  s->pr_q, &s->ds->pcg[0], s->pr_k);
        return;
    }
    VDISPATCH(s, WLK_RESTRICT, l > 0, lc.vt, k_restrict_r<2>, k_restrict_r<3>, lf.g, lc.g, lc.vt, lc.plain, lf.r, lc.iD, lc.r, lc.x, &s->ds->pcg[l + 1], s->rb);
}

void wl_k_prolong(wl_sim* s, int l)
{
    Level &lf = s->lev[l], &lc = s->lev[l + 1];
    if (l >= s->pk_level) { CoarseProg P; P.n = 0; prog_add(P, COP_PROLONG, l, 0); coarse_launch(s, P); return; }
    if (l == 0 && s->pr_r) {       // ... and is applied here, where x and r are rewritten anyway
        const float* rin = s->pr_r;
        s->pr_r = nullptr;
        VDISPATCH(s, WLK_PROLONG, 0, lf.vt, k_prolong_pend<2>, k_prolong_pend<3>, lf.g, lc.g, lf.vt, lf.plain, lf.L, lf.Lc, lf.iD, lc.x, lf.x, lf.r, &s->ds->pcg[0], s->rb,
                  rin, s->pr_e, s->pr_q, s->pr_k);
        return;
    }
    VDISPATCH(s, WLK_PROLONG, l > 0, lf.vt, k_prolong<2>, k_prolong<3>, lf.g, lc.g, lf.vt, lf.plain, lf.L, lf.Lc, lf.iD, lc.x, lf.x, lf.r, &s->ds->pcg[l], s->rb);
}

void wl_k_rsum(wl_sim* s, int l)
{
    Level& lv = s->lev[l];
    VDISPATCH(s, WLK_MISC, l > 0, lv.vt, k_rsum<2>, k_rsum<3>, lv.g, lv.vt, lv.plain, lv.r, lv.iD, &s->ds->pcg[l], s->rb);
}

void wl_k_smooth(wl_sim* s, int l, int iters, int need_r)
{
    Level& lv = s->lev[l];
    if (l >= s->pk_level) { CoarseProg P; P.n = 0; prog_add(P, COP_SMOOTH, l, iters); coarse_launch(s, P); return; }
    if (s->fused && s->fast_A && s->bulk_A && wl_k_smooth_fused(s, l, iters, need_r)) return;
    PcgScal* sc = &s->ds->pcg[l];
    float* ea = lv.e;      // direction written by the running A pass
    float* eb = lv.e2;     // previous direction
    // 3-D levels go through the shared-memory kernel of wl_pcgfast.cu
    const int fast = s->fast_A && wl_pcg_fast_ok(s, l);
    for (int k = 1; k <= iters; ++k) {
        if (fast) wl_k_pcg_A_fast(s, l, k == 1, eb, ea);
        else if (k == 1)
            VDISPATCH(s, WLK_PCG_MATVEC, l > 0, lv.vt, (k_pcg_A<2, 1>), (k_pcg_A<3, 1>), lv.g, lv.vt, lv.plain, lv.L, lv.Lc, lv.iDc,
                      eb, lv.r, lv.iD, ea, lv.q, sc, s->rb);
        else
            VDISPATCH(s, WLK_PCG_MATVEC, l > 0, lv.vt, (k_pcg_A<2, 0>), (k_pcg_A<3, 0>), lv.g, lv.vt, lv.plain, lv.L, lv.Lc, lv.iDc,
                      eb, lv.r, lv.iD, ea, lv.q, sc, s->rb);
        VDISPATCH(s, WLK_PCG_UPDATE, l > 0, lv.vt, k_pcg_B<2>, k_pcg_B<3>, lv.g, lv.vt, lv.plain, lv.Lc, lv.iDc, lv.x, lv.r, ea, lv.q, lv.iD, sc, s->rb,
                  k == 1 ? 1 : 0, k == iters ? 1 : 0);
        float* t = ea; ea = eb; eb = t;
    }
    cudaMemsetAsync(&sc->rsum, 0, sizeof(double), s->st);    // the mean of r has been removed (R-T2)
}

// V-cycle below level l (R-S): restrict l -> l+1; V-cycle(l+1); smooth(l+1); prolong l+1 -> l.
// From level pk_level on, the whole remaining chain is one k_coarse launch.
void wl_k_vcycle(wl_sim* s, int l)
{
    if (l + 1 >= s->nlev) return;
    const int it = s->cfg.mg.smooth_iters;
    if (l >= s->pk_level) {         // stage hook on a coarse level: the sub-V-cycle as one program
        CoarseProg P; P.n = 0;
        for (int j = l; j <= s->nlev - 2; ++j) prog_add(P, COP_RESTRICT, j, 0);
        for (int j = s->nlev - 1; j > l; --j) { prog_add(P, COP_SMOOTH, j, it); prog_add(P, COP_PROLONG, j - 1, 0); }
        coarse_launch(s, P);
        return;
    }
    wl_k_restrict(s, l);
    if (l + 1 >= s->pk_level) {
        const int a = l + 1;
        CoarseProg P; P.n = 0;
        for (int j = a; j <= s->nlev - 2; ++j) prog_add(P, COP_RESTRICT, j, 0);
        for (int j = s->nlev - 1; j >= a; --j) { prog_add(P, COP_SMOOTH, j, it); if (j > a) prog_add(P, COP_PROLONG, j - 1, 0); }
        coarse_launch(s, P);
    } else {
        if (l + 1 < s->nlev - 1) wl_k_vcycle(s, l + 1);
        wl_k_smooth(s, l + 1, it, 0);       // the prolongation reads x of the coarse level only
    }
    wl_k_prolong(s, l);
}

void wl_k_resmax(wl_sim* s)
{
    Level& lv = s->lev[0];
    Tiling T = wl_tiles_interior(s, lv.g);
    DISPATCH(s, WLK_RESMAX, 0, k_resmax, T, lv.g, T, lv.r, s->ds, s->rb);
}
