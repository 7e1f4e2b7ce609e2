// wl_pcgfused.cu -- the Jacobi-PCG smoother (DESIGN.md R-T, R-T2) with ONE sweep per iteration.
//
// The two-pass form (wl_pcgfast.cu pass A, k_pcg_B) needs rho' = r'.(iD r') of the updated residual r' = r - alpha q
// before it can form the next direction, hence a second sweep.  But
//     rho' = rho - 2 alpha (q . iD r) + alpha^2 (q . iD q),
// so a sweep that also accumulates q.iD r and q.iD q knows alpha AND beta when it ends, and the update of iteration k
// can ride on the sweep of iteration k+1:
//     first sweep  (k_pcg_fused<1>):             e' = iD (r - m); q = A e'; gamma, rho, q.iD(r-m), q.iD q
//     fused sweep  (k_pcg_fused<0>, iterations 2..n): r' = (r - m) - alpha q [r and q with halos]; x += alpha e;
//                                                  e' = beta e + iD r'; q' = A e'; gamma, q'.iD r', q'.iD q'
//     last sweep   (k_pcg_last, pointwise):       x += alpha e; r' = r - alpha q  (x alone where nobody reads r' any more)
// 12 + 32 (n-1) + 24 bytes per cell instead of 12 + 16 (n-1) + 24 n, n + 1 launches instead of 2 n.  r and q ping-pong
// between two buffers (a block reads the OLD r and q of its neighbours' cells); the last sweep writes r back to where it
// was, and a sweep that finds the smoother stopped applies the update still owed or copies r across, so after the call r
// is where it was.  The planes of r, e, q (with halos) and x (own cells) arrive as TMA boxes, three planes ahead of use.
// A TMA box cannot wrap, so on a level that is periodic in x or y the arrays read with halos (r, e, q) carry periodic GHOST cells:
// whoever writes cell 1 / n of a periodic direction also writes the ghost n+1 / 0 (the sweeps do it for r', e', q'; a small kernel
// does it for r before the first sweep, since r comes from the residual / restriction / prolongation kernels, which wrap at load
// time and keep no ghosts).  z wraps through the plane coordinate of the box.
// Levels this form does not take (fewer than 68 cells along x, 2-D) keep the two-pass form.
#include <cstdio>
#include <cstring>
#include "wl_internal.h"
#include "wl_tma.cuh"

#define FF_S 3                    // raw stages
#define FF_BPS 2                  // resident blocks per SM of a fused sweep (the first sweep, with a third of the shared memory, runs 3)
#define FF_RW 136                 // floats per shared row: cells x0-4 .. x0+131
#define FF_PL (FF_RW * 10)        // floats per shared plane: rows y0-1 .. y0+8
#define FF_PLR ((FF_PL + 31) / 32 * 32)
#define FF_XB 1024                // floats of the x box of a plane: the tile's own 128 x 8 cells

__device__ __forceinline__ int ff_src(int c, int n, int per)
{
    if (per) { if (c < 1) c += n; else if (c > n) c -= n; }
    return c < 0 ? 0 : (c > n + 1 ? n + 1 : c);
}
__device__ __forceinline__ int ff_bnd(int c, int n, int per) { return (!per && (c == 1 || c == n)) ? 1 : 0; }
struct FfTab { float t0, t1, t2, t3; };
__device__ __forceinline__ float ff_pick(const FfTab& T, int n) { return n == 0 ? T.t0 : (n == 1 ? T.t1 : (n == 2 ? T.t2 : T.t3)); }

// r' and e' at one position: r' = (r - m [coupled cells only]) - alpha q ; e' = beta e + iD r'
__device__ __forceinline__ float ff_rnew(float rr, float qq, float d, float alpha, float m)
{
    float t = rr;
    if (m != 0.0f && d != 0.0f) t -= m;
    return __fmaf_rn(-alpha, qq, t);
}
__device__ __forceinline__ float ff_dir(float ee, float rn, float d, float beta) { return __fmaf_rn(beta, ee, __fmul_rn(d, rn)); }

// One tile of a sweep.  FIRST: the first iteration (r only is staged; nothing is updated).  Otherwise r, e and q of the
// previous iteration are staged (one TMA box each per plane, halos included), r' and e' are formed at every position of
// the plane, r' and x are stored for the tile's own cells, and the stencil runs on e' as in wl_pcgfast.cu.
// acc: gamma = q'.e', q'.(iD r'), q'.(iD q'), and (FIRST) rho = e'.(r - m).
template <int FIRST, int MODE, int PER>
__device__ __forceinline__ void ff_tile(const Grid& g, const VT& vt, int tile, float Lc, float iDc, const FfTab& T, float alpha, float beta, float m,
                                        const float* __restrict__ L, const float* __restrict__ iD, float* __restrict__ x, float* __restrict__ rout,
                                        float* __restrict__ eout, float* __restrict__ qout, float* raw, float* ebuf, double (&acc)[4],
                                        unsigned mbar, unsigned& phases, const CUtensorMap* tm_r, const CUtensorMap* tm_e, const CUtensorMap* tm_q, const CUtensorMap* tm_x)
{
    constexpr bool PLB = MODE == TM_PLB, GEN = MODE == TM_GEN;
    constexpr int NA = FIRST ? 1 : 3;
    constexpr int LX = 32, LY = 8, RW = FF_RW, PL = FF_PL, PLR = FF_PLR, SP = NA * PLR + (FIRST ? 0 : FF_XB);
    const int tid = threadIdx.x, tx = tid & (LX - 1), ty = tid >> 5;
    const int tix = tile % vt.ntx, rem = tile / vt.ntx, tiy = rem % vt.nty, tiz = rem / vt.nty;
    const int x0 = 1 + 4 * LX * tix, y0 = 1 + LY * tiy;
    const int z0 = 1 + tiz * vt.zc, z1 = min(z0 + vt.zc - 1, g.n[2]);
    // every other slab of tiles is marched downwards: a tile and its z neighbours then read the planes they share at the
    // same time (both at their start, or both at their end), and the second reader finds them in L2
    const int dir = (tiz & 1) ? -1 : 1, zs = dir > 0 ? z0 : z1;
    const int gx = tix * LX + tx, c0 = 1 + 4 * gx, c1 = y0 + ty;
    // the last tile of a row may stick out in x and y: positions past the row read zeros (the pad of the array, or the zero
    // fill of the TMA box), form finite values nobody uses, and store nothing; n0 % 4 == 0: whole groups only
    const bool own = gx < vt.ngx, valid = own && c1 <= g.n[1];
    const int sy = (int)g.sy, sz = (int)g.sz;
    const int off_own = WL_OFF + c0 + ff_src(c1, g.n[1], 0) * sy;
    // 1/D keeps no ghosts: where a thread's group stands on a periodic ghost (the first group past a ragged row end in x, the row
    // past the last one in y) it takes 1/D of the cells the ghosts mirror
    const int px = PER ? g.per[0] : 0, py = PER ? g.per[1] : 0;       // PER == 0: the level wraps in neither x nor y
    const bool wrapx = px && c0 == g.n[0] + 1;
    const int off_d = WL_OFF + (wrapx ? 1 : c0) + ff_src(c1, g.n[1], py) * sy;
    const int idx_own = (ty + 1) * RW + 4 + 4 * tx;
    bool hrow = false, hrow_ld = false; int off_h = 0, idx_h = 0, hc0 = 0, hc1 = 0;
    if (tid < 2 * LX) {
        const int hr = tid >> 5, hx = tid & (LX - 1);
        hrow = true; hrow_ld = tix * LX + hx < vt.ngx;
        hc0 = 1 + 4 * (tix * LX + hx); hc1 = hr ? y0 + LY : y0 - 1;
        off_h = WL_OFF + hc0 + ff_src(hc1, g.n[1], py) * sy;        // 1/D keeps no ghosts: the wrapped row
        idx_h = (hr ? LY + 1 : 0) * RW + 4 + 4 * hx;
    }
    bool hcol = false; int off_x = 0, idx_x = 0, xc0 = 0, xc1 = 0;
    if (tid >= 64 && tid < 64 + 2 * LY) {     // not the threads that already form the halo rows
        const int rr = (tid - 64) >> 1, side = tid & 1;
        hcol = true;
        xc0 = side ? x0 + 4 * LX : x0 - 1; xc1 = y0 + rr;
        off_x = WL_OFF + ff_src(xc0, g.n[0], px) + ff_src(xc1, g.n[1], 0) * sy;
        idx_x = (rr + 1) * RW + (side ? 4 + 4 * LX : 3);
    }
    // periodic ghosts of the arrays written here (see the head of the file): cell 1 -> ghost n+1, cell n -> ghost 0, per direction
    const bool gx_lo = px && c0 == 1, gx_hi = px && c0 + 3 == g.n[0];
    const bool gy_lo = py && c1 == 1, gy_hi = py && c1 == g.n[1];
    auto ghosts = [&](float* __restrict__ a, int i, const float4& v) {
        if (!PER) return;
        if (gx_lo) a[i + g.n[0]] = v.x;
        if (gx_hi) a[i - c0] = v.w;
        if (gy_lo) *reinterpret_cast<float4*>(a + i + g.n[1] * sy) = v;
        if (gy_hi) *reinterpret_cast<float4*>(a + i - g.n[1] * sy) = v;
    };
    const unsigned sraw = (unsigned)__cvta_generic_to_shared(raw);
    auto issue = [&](int p, int slot) {
        if (p >= z0 - 1 && p <= z1 + 1 && tid == 0) {
            const unsigned bar = mbar + 8u * (unsigned)slot;
            const unsigned dst = sraw + 4u * (unsigned)(slot * SP);
            const int zc_ = ff_src(p, g.n[2], g.per[2]);
            const bool inner = !FIRST && p >= z0 && p <= z1;      // x: the tile's own cells only
            mbar_expect_tx(bar, (unsigned)(NA * PL * 4 + (inner ? FF_XB * 4 : 0)));
            if (inner) tma_box3(dst + 12u * PLR, tm_x, WL_OFF + x0, y0, zc_, bar);
            tma_box3(dst, tm_r, WL_OFF + x0 - 4, y0 - 1, zc_, bar);
            if (!FIRST) {
                tma_box3(dst + 4u * PLR, tm_e, WL_OFF + x0 - 4, y0 - 1, zc_, bar);
                tma_box3(dst + 8u * PLR, tm_q, WL_OFF + x0 - 4, y0 - 1, zc_, bar);
            }
        }
    };
    auto arrived = [&](int slot) {
        mbar_wait(mbar + 8u * (unsigned)slot, (phases >> slot) & 1u);
        phases ^= 1u << slot;
    };
    // ---- analytic coefficients and 1/D of this thread's cells (without the z part)
    float cxl[4], cxh[4], cyl = Lc, cyh = Lc;
    float d_in[4], d_bz[4], dh_in[4], dh_bz[4], dx_in = iDc, dx_bz = iDc;
#pragma unroll
    for (int k = 0; k < 4; ++k) { cxl[k] = Lc; cxh[k] = Lc; d_in[k] = iDc; d_bz[k] = iDc; dh_in[k] = iDc; dh_bz[k] = iDc; }
    if (PLB) {
        const int byo = ff_bnd(c1, g.n[1], py), byh = ff_bnd(hc1, g.n[1], py);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (!px && c0 + k == 1) cxl[k] = 0.0f;
            if (!px && c0 + k == g.n[0]) cxh[k] = 0.0f;
            const int bo = byo + ff_bnd(c0 + k, g.n[0], px), bh = byh + ff_bnd(hc0 + k, g.n[0], px);
            d_in[k] = ff_pick(T, bo); d_bz[k] = ff_pick(T, bo + 1);
            dh_in[k] = ff_pick(T, bh); dh_bz[k] = ff_pick(T, bh + 1);
        }
        if (!py && c1 == 1) cyl = 0.0f;
        if (!py && c1 == g.n[1]) cyh = 0.0f;
        const int bx = ff_bnd(xc0, g.n[0], px) + ff_bnd(xc1, g.n[1], py);
        dx_in = ff_pick(T, bx); dx_bz = ff_pick(T, bx + 1);
    }
    auto load_iD = [&](int p, bool full) {    // GEN: 1/D of plane p at the positions the operands come from
        const int zo = ff_src(p, g.n[2], g.per[2]) * sz;
        if (own || wrapx) unpack4(ld4(iD, off_d + zo), d_in);
        if (full && hrow_ld) unpack4(ld4(iD, off_h + zo), dh_in);
        if (full && hcol) dx_in = ld1(iD, off_x + zo);
    };
    // GEN: L and 1/D are plain loads, consumed in the iteration that issues them; what the next iterations will load is pulled into
    // L2 a plane (L) or two (1/D) ahead, so that those loads wait for L2 and not for DRAM
    auto pf = [](const float* a) { asm volatile("prefetch.global.L2 [%0];" ::"l"(a)); };
    auto prefetch_gen = [&](int pd, int pl) {
        const int zo = ff_src(pd, g.n[2], g.per[2]) * sz;
        if (own || wrapx) pf(iD + off_d + zo);
        if (hrow_ld) pf(iD + off_h + zo);
        if (hcol) pf(iD + off_x + zo);
        if (valid && pl >= z0 && pl <= z1) {
            const int i = off_own + pl * sz;
            pf(L + i); if (tx == LX - 1) pf(L + i + 4);
            pf(L + g.nalloc + i); if (ty == LY - 1) pf(L + g.nalloc + i + sy);
            pf(L + 2 * g.nalloc + i + (dir > 0 ? sz : 0));
        }
    };
    // plane p from stage slot `slot`: r' and x stored for the own cells, e' -> registers and shared, iD r' and iD -> registers
    auto form = [&](int p, int slot, float (&ep)[4], float (&zr)[4], float (&dd)[4], bool full) {
        const float* st = raw + slot * SP;
        float* eb = ebuf + (p & 1) * PL;
        const bool bz = PLB && ff_bnd(p, g.n[2], g.per[2]);     // block-uniform
        {
            float rr[4], ee[4] = { 0.f, 0.f, 0.f, 0.f }, qv[4] = { 0.f, 0.f, 0.f, 0.f }, rn[4];
            unpack4(*reinterpret_cast<const float4*>(st + idx_own), rr);
            if (!FIRST) { unpack4(*reinterpret_cast<const float4*>(st + PLR + idx_own), ee); unpack4(*reinterpret_cast<const float4*>(st + 2 * PLR + idx_own), qv); }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float d = bz ? d_bz[k] : d_in[k];
                rn[k] = FIRST ? rr[k] - m : ff_rnew(rr[k], qv[k], d, alpha, m);
                zr[k] = __fmul_rn(d, rn[k]);
                ep[k] = FIRST ? zr[k] : __fmaf_rn(beta, ee[k], zr[k]);
                dd[k] = d;
            }
            if (valid && p >= z0 && p <= z1) {
                if (FIRST) {
                    float sr = ep[0] * rn[0];
                    sr = __fmaf_rn(ep[1], rn[1], sr); sr = __fmaf_rn(ep[2], rn[2], sr); sr = __fmaf_rn(ep[3], rn[3], sr);
                    acc[3] += (double)sr;
                } else {
                    const int i = off_own + p * sz;
                    float xv[4];
                    unpack4(*reinterpret_cast<const float4*>(st + 3 * PLR + 128 * ty + 4 * tx), xv);
                    const float4 rv = make_float4(rn[0], rn[1], rn[2], rn[3]);
                    *reinterpret_cast<float4*>(rout + i) = rv;
                    ghosts(rout, i, rv);
                    *reinterpret_cast<float4*>(x + i) = make_float4(xv[0] + alpha * ee[0], xv[1] + alpha * ee[1], xv[2] + alpha * ee[2], xv[3] + alpha * ee[3]);
                }
            }
        }
        if (!full) return;
        *reinterpret_cast<float4*>(eb + idx_own) = make_float4(ep[0], ep[1], ep[2], ep[3]);
        if (hrow) {
            float rr[4], ee[4] = { 0.f, 0.f, 0.f, 0.f }, qv[4] = { 0.f, 0.f, 0.f, 0.f }, eh[4];
            unpack4(*reinterpret_cast<const float4*>(st + idx_h), rr);
            if (!FIRST) { unpack4(*reinterpret_cast<const float4*>(st + PLR + idx_h), ee); unpack4(*reinterpret_cast<const float4*>(st + 2 * PLR + idx_h), qv); }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float d = bz ? dh_bz[k] : dh_in[k];
                const float rn = FIRST ? rr[k] - m : ff_rnew(rr[k], qv[k], d, alpha, m);
                eh[k] = FIRST ? __fmul_rn(d, rn) : ff_dir(ee[k], rn, d, beta);
            }
            *reinterpret_cast<float4*>(eb + idx_h) = make_float4(eh[0], eh[1], eh[2], eh[3]);
        }
        if (hcol) {
            const float d = bz ? dx_bz : dx_in;
            const float rr = st[idx_x];
            const float rn = FIRST ? rr - m : ff_rnew(rr, st[2 * PLR + idx_x], d, alpha, m);
            eb[idx_x] = FIRST ? __fmul_rn(d, rn) : ff_dir(st[PLR + idx_x], rn, d, beta);
        }
    };

    __syncthreads();                          // the previous tile's shared planes are no longer read
    // ---- prologue: the plane before the first one (own column only) in slot FF_S-1, the first one (full) in slot 0
    float zm[4], zc[4], zp[4], zrc[4], zrp[4], dc[4], dp[4], dummy[4], dummy2[4];
    issue(zs - dir, FF_S - 1);
    issue(zs, 0);
    issue(zs + dir, 1);
    if (GEN) { load_iD(zs - dir, false); prefetch_gen(zs, zs); prefetch_gen(zs + dir, zs); }
    arrived(FF_S - 1);
    form(zs - dir, FF_S - 1, zm, dummy, dummy2, false);
    if (GEN) load_iD(zs, true);
    arrived(0);
    form(zs, 0, zc, zrc, dc, true);
    __syncthreads();                          // slot FF_S-1 is free again
#pragma unroll
    for (int d = 2; d < FF_S; ++d) issue(zs + d * dir, d);
    int sl = 0;                               // slot of plane z
    for (int n = z1 - z0, z = zs; n >= 0; --n, z += dir) {
        const int sn = sl + 1 == FF_S ? 0 : sl + 1;       // slot of the plane after z
        float lx[5] = { 0.f, 0.f, 0.f, 0.f, 0.f }, ly[4] = { 0.f, 0.f, 0.f, 0.f }, lyp[4] = { 0.f, 0.f, 0.f, 0.f };
        float lz[4] = { 0.f, 0.f, 0.f, 0.f }, lzp[4] = { 0.f, 0.f, 0.f, 0.f };
        if (GEN) {                            // 1/D of the next plane and the face coefficients of the own cells of plane z
            prefetch_gen(z + 2 * dir, z + dir);
            load_iD(z + dir, true);
            if (valid) {
                const int i = off_own + z * sz;
                const float4 a = ld4(L, i);
                lx[0] = a.x; lx[1] = a.y; lx[2] = a.z; lx[3] = a.w; lx[4] = ld1(L, i + 4);
                unpack4(ld4(L + g.nalloc, i), ly); unpack4(ld4(L + g.nalloc, i + sy), lyp);
                unpack4(ld4(L + 2 * g.nalloc, i), lz); unpack4(ld4(L + 2 * g.nalloc, i + sz), lzp);
            }
        }
        arrived(sn);
        __syncthreads();                      // e'(z) in shared is complete; the slot of plane z is free
        issue(z + FF_S * dir, sl);
        form(z + dir, sn, zp, zrp, dp, true);
        // stencil at plane z
        const float* eb = ebuf + (z & 1) * PL;
        const float4 ym = *reinterpret_cast<const float4*>(eb + idx_own - RW);
        const float4 yp = *reinterpret_cast<const float4*>(eb + idx_own + RW);
        float xm = __shfl_up_sync(0xffffffffu, zc[3], 1), xp = __shfl_down_sync(0xffffffffu, zc[0], 1);
        if (tx == 0) xm = eb[idx_own - 1];
        if (tx == LX - 1) xp = eb[idx_own + 4];
        float czl = Lc, czh = Lc;
        if (PLB) { if (!g.per[2] && z == 1) czl = 0.0f; if (!g.per[2] && z == g.n[2]) czh = 0.0f; }
        const float w[6] = { xm, zc[0], zc[1], zc[2], zc[3], xp };
        const float ymv[4] = { ym.x, ym.y, ym.z, ym.w }, ypv[4] = { yp.x, yp.y, yp.z, yp.w };
        float qq[4], zlo[4], zhi[4];          // the planes below and above z, whichever way the march goes
#pragma unroll
        for (int k = 0; k < 4; ++k) { zlo[k] = dir > 0 ? zm[k] : zp[k]; zhi[k] = dir > 0 ? zp[k] : zm[k]; }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float ec = w[k + 1];
            float a = 0.0f;
            if (GEN) {
                a += lx[k + 1] * (w[k + 2] - ec) - lx[k] * (ec - w[k]);
                a += lyp[k] * (ypv[k] - ec) - ly[k] * (ec - ymv[k]);
                a += lzp[k] * (zhi[k] - ec) - lz[k] * (ec - zlo[k]);
            } else {
                a += cxh[k] * (w[k + 2] - ec) - cxl[k] * (ec - w[k]);
                a += cyh * (ypv[k] - ec) - cyl * (ec - ymv[k]);
                a += czh * (zhi[k] - ec) - czl * (ec - zlo[k]);
            }
            qq[k] = a;
        }
        if (valid) {
            const int i = off_own + z * sz;
            const float4 ev = make_float4(zc[0], zc[1], zc[2], zc[3]), qv = make_float4(qq[0], qq[1], qq[2], qq[3]);
            *reinterpret_cast<float4*>(eout + i) = ev;
            *reinterpret_cast<float4*>(qout + i) = qv;
            ghosts(eout, i, ev);
            ghosts(qout, i, qv);
            // fp32 products summed over the thread's four cells, accumulated in fp64 once per plane
            float sg = qq[0] * zc[0], s2 = qq[0] * zrc[0], s3 = qq[0] * __fmul_rn(dc[0], qq[0]);
#pragma unroll
            for (int k = 1; k < 4; ++k) {
                sg = __fmaf_rn(qq[k], zc[k], sg); s2 = __fmaf_rn(qq[k], zrc[k], s2); s3 = __fmaf_rn(qq[k], __fmul_rn(dc[k], qq[k]), s3);
            }
            acc[0] += (double)sg; acc[1] += (double)s2; acc[2] += (double)s3;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) { zm[k] = zc[k]; zc[k] = zp[k]; zrc[k] = zrp[k]; dc[k] = dp[k]; }
        sl = sn;
    }
}

// The update of one iteration alone, on one tile: x += alpha e; rout = (rin - m) - alpha q  (UPDATE), or rout = rin (the
// smoother has stopped and r only has to change buffers), or (UPDATE == 2) x += alpha e alone.  Pointwise: no halos, plain loads.
template <int UPDATE>
__device__ __forceinline__ void ff_pointwise(const Grid& g, const VT& vt, int tile, int mode, float alpha, float m, const float* __restrict__ iD,
                                             float* __restrict__ x, const float* rin, float* rout,
                                             const float* __restrict__ e, const float* __restrict__ q)
{
    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
    const int tix = tile % vt.ntx, rem = tile / vt.ntx, tiy = rem % vt.nty, tiz = rem / vt.nty;
    const int c0 = 1 + 4 * (tix * 32 + tx), c1 = 1 + 8 * tiy + ty;
    const int z0 = 1 + tiz * vt.zc, z1 = min(z0 + vt.zc - 1, g.n[2]);
    if (c1 > g.n[1] || c0 > g.n[0]) return;
    const int off = WL_OFF + c0 + c1 * (int)g.sy;
    for (int z = z0; z <= z1; ++z) {
        const int i = off + z * (int)g.sz;
        if (UPDATE == 2) {
            float xv[4], ee[4];
            unpack4(*reinterpret_cast<const float4*>(x + i), xv);
            unpack4(ld4(e, i), ee);
            *reinterpret_cast<float4*>(x + i) = make_float4(xv[0] + alpha * ee[0], xv[1] + alpha * ee[1], xv[2] + alpha * ee[2], xv[3] + alpha * ee[3]);
            continue;
        }
        float rr[4];
        unpack4(*reinterpret_cast<const float4*>(rin + i), rr);
        if (UPDATE) {
            float xv[4], ee[4], qv[4], dd[4] = { 1.f, 1.f, 1.f, 1.f };
            unpack4(*reinterpret_cast<const float4*>(x + i), xv);
            unpack4(ld4(e, i), ee); unpack4(ld4(q, i), qv);
            if (m != 0.0f && mode == TM_GEN) unpack4(ld4(iD, i), dd);     // body-free tiles: every cell is coupled
#pragma unroll
            for (int k = 0; k < 4; ++k) { rr[k] = ff_rnew(rr[k], qv[k], dd[k], alpha, m); xv[k] += alpha * ee[k]; }
            *reinterpret_cast<float4*>(x + i) = make_float4(xv[0], xv[1], xv[2], xv[3]);
        }
        *reinterpret_cast<float4*>(rout + i) = make_float4(rr[0], rr[1], rr[2], rr[3]);
    }
}

// kprev: the iteration whose update (alpha, and the mean m when kprev == 1) this sweep applies; 0 in the first sweep
// PER: the level wraps in x or y (ghost cells maintained, 1/D taken from the mirrored cells); 0 keeps all of that out of the code
template <int FIRST, int PER>
__global__ void __launch_bounds__(WL_VB, FIRST ? 3 : FF_BPS) k_pcg_fused(Grid g, VT vt, const int* __restrict__ plain, const int* __restrict__ sched, float Lc, float iDc, int kprev,
                                                         const float* __restrict__ L, const float* __restrict__ iD, float* __restrict__ x,
                                                         const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ ein,
                                                         float* __restrict__ eout, const float* __restrict__ qin, float* __restrict__ qout,
                                                         PcgScal* sc, RedBuf rb, const __grid_constant__ CUtensorMap tm_r,
                                                         const __grid_constant__ CUtensorMap tm_e, const __grid_constant__ CUtensorMap tm_q,
                                                         const __grid_constant__ CUtensorMap tm_x)
{
    extern __shared__ __align__(128) float4 ff_smem4[];
    float* sm = reinterpret_cast<float*>(ff_smem4);
    const float mean = sc->nlive > 0.0 ? (float)(sc->rsum / sc->nlive) : 0.0f;
    const float m = (FIRST || kprev == 1) ? mean : 0.0f;
    const float alpha = FIRST ? 0.0f : (float)sc->alpha, beta = FIRST ? 0.0f : (float)sc->beta;
    if (!FIRST && !sc->live) {                // stopped (uniform across the grid: written by an earlier kernel)
        const bool flush = sc->stop_k == kprev;           // the update of the iteration that met the criterion is still owed
        if (!flush && rin == rout) return;
        for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
            if (flush) ff_pointwise<1>(g, vt, tile, plain[tile], alpha, m, iD, x, rin, rout, ein, qin);
            else       ff_pointwise<0>(g, vt, tile, plain[tile], alpha, m, iD, x, rin, rout, ein, qin);
        }
        return;
    }
    constexpr int NA = FIRST ? 1 : 3;
    constexpr int SP = NA * FF_PLR + (FIRST ? 0 : FF_XB);
    float* raw = sm;                          // [FF_S][SP]: r (+ e, q with halos, x without)
    float* ebuf = sm + FF_S * SP;             // [2][FF_PL]
    const unsigned mbar = (unsigned)__cvta_generic_to_shared(sm + FF_S * SP + 2 * FF_PL);
    unsigned phases = 0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < FF_S; ++k) mbar_init(mbar + 8u * k, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    FfTab T;
    T.t0 = 1.0f / (-6.0f * Lc); T.t1 = 1.0f / (-5.0f * Lc); T.t2 = 1.0f / (-4.0f * Lc); T.t3 = 1.0f / (-3.0f * Lc);
    double acc[4] = { 0.0, 0.0, 0.0, 0.0 };
    // tiles in the order of k_tile_sched (wl_poisson.cu): entry = tile | mode << 24, fetched a tile ahead of its use
    int next = blockIdx.x < vt.ntiles ? sched[blockIdx.x] : 0;
    for (int k = blockIdx.x; k < vt.ntiles; k += gridDim.x) {
        const int tile = next & 0xffffff, mode = next >> 24;          // block-uniform
        next = k + gridDim.x < vt.ntiles ? sched[k + gridDim.x] : 0;
#define FF_CALL(M) ff_tile<FIRST, M, PER>(g, vt, tile, Lc, iDc, T, alpha, beta, m, L, iD, x, rout, eout, qout, raw, ebuf, acc, mbar, phases, &tm_r, &tm_e, &tm_q, &tm_x)
        if (mode == TM_PLI) FF_CALL(TM_PLI);
        else if (mode == TM_PLB) FF_CALL(TM_PLB);
        else FF_CALL(TM_GEN);
#undef FF_CALL
    }
    if (grid_reduce<4, OpSum>(acc, rb)) {
        if (threadIdx.x == 0) {
            // alpha of this iteration, and rho' = r'.(iD r') of the residual the NEXT sweep will form, from the recurrence
            const double gamma = acc[0], s2 = acc[1], s3 = acc[2];
            double rho = sc->rho;
            int live = 1;
            if (FIRST) {
                rho = acc[3];
                sc->rho = rho; sc->rho0 = rho; sc->beta = 0.0; sc->stop_k = 0;
                live = fabs(rho) < WL_TAU ? 0 : 1;
            }
            sc->gamma = gamma;
            if (gamma == 0.0 || !isfinite(gamma) || !live) { sc->live = 0; sc->alpha = 0.0; }
            else {
                const double a = rho / gamma;
                const double rho2 = rho - 2.0 * a * s2 + a * a * s3;
                sc->alpha = a;
                if (fabs(rho2) < WL_TAU || fabs(rho2) < WL_THETA * fabs(sc->rho0)) { sc->live = 0; sc->stop_k = kprev + 1; }
                else { sc->live = 1; sc->beta = rho2 / rho; sc->rho = rho2; }
            }
        }
    }
}

// the update of the last iteration (kprev), or what a stopped smoother still owes
__global__ void __launch_bounds__(WL_VB, 4) k_pcg_last(Grid g, VT vt, const int* __restrict__ plain, int kprev, const float* __restrict__ iD, float* __restrict__ x,
                                                       const float* rin, float* rout, const float* __restrict__ e,
                                                       const float* __restrict__ q, const PcgScal* sc, int need_r)
{
    const float m = kprev == 1 && sc->nlive > 0.0 ? (float)(sc->rsum / sc->nlive) : 0.0f;
    const float alpha = (float)sc->alpha;
    const bool update = sc->live || sc->stop_k == kprev;
    if (!update && (rin == rout || !need_r)) return;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        if (update && need_r) ff_pointwise<1>(g, vt, tile, plain[tile], alpha, m, iD, x, rin, rout, e, q);
        else if (update)      ff_pointwise<2>(g, vt, tile, plain[tile], alpha, m, iD, x, rin, rout, e, q);
        else                  ff_pointwise<0>(g, vt, tile, plain[tile], alpha, m, iD, x, rin, rout, e, q);
    }
}

static size_t ff_smem(int first) { return sizeof(float) * ((size_t)FF_S * (first ? FF_PLR : 3 * FF_PLR + FF_XB) + 2 * FF_PL) + 8 * FF_S + 8; }

// 3-D, whole float4 groups and at least 17 of them per row (32 threads along x), 32-bit offsets
int wl_pcg_fused_shape(int nd, const Grid& g, const VT& vt)
{
    return nd == 3 && g.n[0] % 4 == 0 && vt.lxl == 5 && g.nalloc < ((int64_t)1 << 31);
}

// periodic ghost cells of one scalar array in x and y (interior rows / columns only: the stencil needs no corners)
__global__ void k_wrap_ghosts(Grid g, float* __restrict__ a)
{
    const int64_t nx = g.per[0] ? (int64_t)g.n[1] * g.n[2] : 0, ny = g.per[1] ? (int64_t)g.n[0] * g.n[2] : 0;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < nx + ny; t += (int64_t)gridDim.x * blockDim.x) {
        if (t < nx) {
            const int c1 = 1 + (int)(t % g.n[1]), c2 = 1 + (int)(t / g.n[1]);
            const int64_t row = gidx(g, 0, c1, c2);
            a[row] = a[row + g.n[0]];
            a[row + g.n[0] + 1] = a[row + 1];
        } else {
            const int64_t u = t - nx;
            const int c0 = 1 + (int)(u % g.n[0]), c2 = 1 + (int)(u / g.n[0]);
            a[gidx(g, c0, 0, c2)] = a[gidx(g, c0, g.n[1], c2)];
            a[gidx(g, c0, g.n[1] + 1, c2)] = a[gidx(g, c0, 1, c2)];
        }
    }
}

// The smoother on level l as iters + 1 sweeps (see the head of this file).  Returns 0 when the level does not take this form.
int wl_k_smooth_fused(wl_sim* s, int l, int iters, int need_r)
{
    Level& lv = s->lev[l];
    if (!lv.r2 || !lv.q2 || !lv.sched || iters < 1) return 0;
    PcgScal* sc = &s->ds->pcg[l];
    // persistent grids: FF_BPS blocks per SM for the fused sweeps (registers: no spills at 128), 3 for the first sweep
    int grid = lv.vt.ntiles < s->sm_count * FF_BPS ? lv.vt.ntiles : s->sm_count * FF_BPS;
    int grid1 = lv.vt.ntiles < s->sm_count * 3 ? lv.vt.ntiles : s->sm_count * 3;
    if (grid > WL_MAX_PARTIALS) grid = WL_MAX_PARTIALS;
    if (grid1 > WL_MAX_PARTIALS) grid1 = WL_MAX_PARTIALS;
    if (!(s->cd_attr_set & 16)) {         // per handle: a process may hold handles on several devices
        cudaFuncSetAttribute(k_pcg_fused<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ff_smem(1));
        cudaFuncSetAttribute(k_pcg_fused<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ff_smem(1));
        cudaFuncSetAttribute(k_pcg_fused<0, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ff_smem(0));
        cudaFuncSetAttribute(k_pcg_fused<0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ff_smem(0));
        s->cd_attr_set |= 16;
    }
    const bool per = lv.g.per[0] || lv.g.per[1];
    float *ra = lv.r, *rb = lv.r2;            // ra: the residual as it stands
    float *ea = lv.e2, *eb = lv.e;            // ea: the direction of the previous iteration, eb: the one being written
    float *qa = lv.q2, *qb = lv.q;
    // every map this call needs, encoded once per handle (cached) and checked BEFORE the first launch: a failed encode sends
    // the caller to the two-pass form instead of launching a sweep with a stale map
    const float* halo_arrays[6] = { lv.r, lv.r2, lv.e, lv.e2, lv.q, lv.q2 };
    for (int k = 0; k < 6; ++k)
        if (!wl_tensor_map_cached(s->tmc, halo_arrays[k], lv.g, FF_RW, 10)) return 0;
    const CUtensorMap* ptm_x = wl_tensor_map_cached(s->tmc, lv.x, lv.g, 128, 8);
    if (!ptm_x) return 0;
    CUtensorMap tm_r = *wl_tensor_map_cached(s->tmc, ra, lv.g, FF_RW, 10), tm_e, tm_q, tm_x = *ptm_x;
    memset(&tm_e, 0, sizeof(tm_e)); memset(&tm_q, 0, sizeof(tm_q));
    if (per) {                                 // r comes from kernels that keep no ghosts
        ProfScope ps_(s, WLK_MISC, l > 0);
        const int64_t n = (int64_t)lv.g.n[2] * (lv.g.n[0] + lv.g.n[1]);
        int nb = (int)((n + 255) / 256);
        if (nb > s->sm_count * 4) nb = s->sm_count * 4;
        k_wrap_ghosts<<<nb, 256, 0, s->st>>>(lv.g, ra);
    }
    {
        ProfScope ps_(s, WLK_PCG_MATVEC, l > 0);
        auto kern = per ? k_pcg_fused<1, 1> : k_pcg_fused<1, 0>;
        kern<<<grid1, WL_VB, ff_smem(1), s->st>>>(lv.g, lv.vt, lv.plain, lv.sched, lv.Lc, lv.iDc, 0, lv.L, lv.iD, lv.x, ra, rb, ea, eb, qa, qb, sc, s->rb, tm_r, tm_e, tm_q, tm_x);
    }
    for (int k = 2; k <= iters; ++k) {
        float* t = ea; ea = eb; eb = t;
        t = qa; qa = qb; qb = t;
        tm_r = *wl_tensor_map_cached(s->tmc, ra, lv.g, FF_RW, 10);       // cache hits: encoded and checked above
        tm_e = *wl_tensor_map_cached(s->tmc, ea, lv.g, FF_RW, 10);
        tm_q = *wl_tensor_map_cached(s->tmc, qa, lv.g, FF_RW, 10);
        {
            ProfScope ps_(s, WLK_PCG_FUSED, l > 0);
            auto kern = per ? k_pcg_fused<0, 1> : k_pcg_fused<0, 0>;
            kern<<<grid, WL_VB, ff_smem(0), s->st>>>(lv.g, lv.vt, lv.plain, lv.sched, lv.Lc, lv.iDc, k - 1, lv.L, lv.iD, lv.x, ra, rb, ea, eb, qa, qb, sc, s->rb, tm_r, tm_e, tm_q, tm_x);
        }
        t = ra; ra = rb; rb = t;
    }
    if (need_r == 2 && l == 0 && iters >= 2) {
        // the next V-cycle's restriction reads r and its prolongation rewrites x and r: they apply the update on the fly
        // (restrict: 4 more bytes per cell, prolong: 8, instead of a 24 B/cell sweep); iters >= 2: no mean to remove any more
        s->pr_r = ra; s->pr_q = qb; s->pr_e = eb; s->pr_k = iters;
    } else if (need_r < 0 && l == 0) {
        // nobody but apply_gradient reads x of level 0 now: it adds alpha e on the fly (4 instead of 12 bytes per cell)
        s->pend_e = eb;
        s->pend_k = iters;
    } else {
        // the last update brings r back to lv.r: in place when it is there already
        float* rout = lv.r;
        int g2 = lv.vt.ntiles < s->sm_count * 8 ? lv.vt.ntiles : s->sm_count * 8;
        ProfScope ps_(s, WLK_PCG_UPDATE, l > 0);
        k_pcg_last<<<g2, WL_VB, 0, s->st>>>(lv.g, lv.vt, lv.plain, iters, lv.iD, lv.x, ra, rout, eb, qb, sc, need_r > 0 ? 1 : 0);
    }
    cudaMemsetAsync(&sc->rsum, 0, sizeof(double), s->st);    // the mean of r has been removed (R-T2)
    return 1;
}
