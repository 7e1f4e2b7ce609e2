// wl_pcgfast.cu -- pass A of the Jacobi-PCG smoother (DESIGN.md R-T) on the UNIFORM
// tiles of a 3-D level, staged through shared memory.
//
//   e' = beta e + iD r   (first iteration: e' = iD (r - m), R-T2);   q = A e';   gamma = q.e'
//
// The pass is HBM-bound: per cell it must read e and r and write e' and q (16 bytes) and does ~30
// flops.  What limits the register-marching kernel of wl_poisson.cu is not traffic but latency: 125
// registers, two blocks per SM, every plane waits for its own loads.  Here the operands of a tile
// (128 x 8 cells for 32 x 8 threads, one plane at a time, one halo row / column around it) are
// brought into shared memory three planes ahead of their use -- as ONE TMA box per array and plane
// (cp.async.bulk.tensor.3d on a tensor map of the padded array, completing on an mbarrier per stage)
// where a box is all a plane needs, by per-thread cp.async otherwise (periodic x or y, ragged rows) --
// so ~3 planes x 11 KB per block are in flight without holding registers; e' is formed once per cell
// (and once per halo cell) into a shared plane, and the seven-point stencil reads its y neighbours
// from there, its x neighbours by shuffle and its z neighbours from the thread's own registers.
// Face coefficients and 1/D are analytic (tile modes TM_PLI / TM_PLB, wl_vec.cuh): nothing but e and
// r is loaded.  General tiles (TM_GEN: a body or its one-cell neighbourhood, a few per cent of a
// level) take the same route; they load 1/D and the face coefficients of their own cells before the
// wait for the plane's operands.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include "wl_internal.h"
#include "wl_tma.cuh"

#ifndef WL_FA_MINB
#define WL_FA_MINB 4
#endif
#ifndef FA_S
#define FA_S 3
#endif
                                    // raw stages: planes z+1 .. z+3 in flight while plane z is computed

// cp.async of 16 / 4 bytes; the destination is a 32-bit shared-window address
__device__ __forceinline__ void cp16(unsigned d, const float* gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp4(unsigned d, const float* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// source coordinate of a (possibly halo) coordinate c of a direction with n cells: periodic wrap,
// otherwise the ghost cells 0 and n+1 of the padded array (never written: zero); anything further out
// belongs to idle threads and is clamped to a valid address
__device__ __forceinline__ int fa_src(int c, int n, int per)
{
    if (per) { if (c < 1) c += n; else if (c > n) c -= n; }
    return c < 0 ? 0 : (c > n + 1 ? n + 1 : c);
}
// 1 when cell coordinate c of a non-periodic direction has a boundary face
__device__ __forceinline__ int fa_bnd(int c, int n, int per) { return (!per && (c == 1 || c == n)) ? 1 : 0; }

struct FaTab { float t0, t1, t2, t3; };     // iD of a body-free cell with 0..3 boundary faces
__device__ __forceinline__ float fa_pick(const FaTab& T, int n) { return n == 0 ? T.t0 : (n == 1 ? T.t1 : (n == 2 ? T.t2 : T.t3)); }

template <int FIRST>
__device__ __forceinline__ float fa_dir(float ee, float rr, float d, float beta, float m)
{
    return FIRST ? __fmul_rn(d, rr - m) : __fmaf_rn(beta, ee, __fmul_rn(d, rr));
}

// One tile.  MODE (static): TM_PLB, the tile touches a non-periodic domain boundary and coefficients and 1/D
// depend on the cell position; TM_PLI, they are the constants Lc and iDc; TM_GEN, they are loaded.  Everything that does not depend on the plane is
// computed once per tile; the stage of a plane rotates through FA_S slots without a division.
// BULK (static): an operand plane of the tile (cells x0-4 .. x0+4LX+3 of rows y0-1 .. y0+LY: both halos included) arrives as
// ONE TMA box per array (cp.async.bulk.tensor.3d on a tensor map of the padded array), issued by one thread and completing
// on one mbarrier per stage, instead of one to three cp.async per thread: no per-thread copy instructions or address
// arithmetic.  Requires non-periodic x and y (a box cannot wrap; z wraps through the plane coordinate) and tiles that do not
// stick out of the row.
template <int FIRST, int MODE, int LXL, int BULK>
__device__ __forceinline__ void fa_tile(const Grid& g, const VT& vt, int tile, float Lc, float iDc, const FaTab& T, float beta, float m,
                                        const float* __restrict__ ein, const float* __restrict__ r, const float* __restrict__ L, const float* __restrict__ iD,
                                        float* __restrict__ eout, float* __restrict__ q, float* raw, float* ebuf, double (&acc)[2],
                                        unsigned mbar, unsigned& phases, const CUtensorMap* tm_r, const CUtensorMap* tm_e)
{
    constexpr bool PLB = MODE == TM_PLB, GEN = MODE == TM_GEN;
    constexpr int NA = FIRST ? 1 : 2;
    constexpr int LX = 1 << LXL, LY = WL_VB >> LXL;
    constexpr int RW = 4 * LX + 8, PL = RW * (LY + 2);
    constexpr int PLR = BULK ? (PL + 31) / 32 * 32 : PL;      // raw planes of the TMA path start on 128-byte boundaries
    constexpr int SP = NA * PLR;
    const int tid = threadIdx.x, tx = tid & (LX - 1), ty = tid >> LXL;
    const int tix = tile % vt.ntx, rem = tile / vt.ntx, tiy = rem % vt.nty, tiz = rem / vt.nty;
    const int x0 = 1 + 4 * LX * tix, y0 = 1 + LY * tiy;
    const int z0 = 1 + tiz * vt.zc, z1 = min(z0 + vt.zc - 1, g.n[2]);
    // ---- what this thread copies for every plane (pointers at plane coordinate 0)
    const int gx = tix * LX + tx, c0 = 1 + 4 * gx, c1 = y0 + ty;
    const bool valid = gx < vt.ngx && c1 <= g.n[1];       // n0 % 4 == 0: whole groups only
    // in a tile that sticks out of the row, the group after the last one stands for cells n0+1.. : the wrapped
    // first group of the row (periodic x) or zeros (the ghost cell of a boundary whose face coefficient is 0)
    const bool own = gx < vt.ngx || (g.per[0] && gx == vt.ngx);
    // element offsets fit 32 bits: the host takes this path only for arrays below 2^31 floats
    const int sy = (int)g.sy, sz = (int)g.sz;
    const int off_own = WL_OFF + (gx < vt.ngx ? c0 : 1) + fa_src(c1, g.n[1], g.per[1]) * sy;
    const int idx_own = (ty + 1) * RW + 4 + 4 * tx;
    bool hrow = false; int off_h = 0, idx_h = 0, hc0 = 0, hc1 = 0;
    if (tid < 2 * LX) {
        const int hr = tid >> LXL, hx = tid & (LX - 1), gxh = tix * LX + hx;
        hrow = gxh < vt.ngx;
        hc0 = 1 + 4 * gxh; hc1 = hr ? y0 + LY : y0 - 1;
        off_h = WL_OFF + hc0 + fa_src(hc1, g.n[1], g.per[1]) * sy;
        idx_h = (hr ? LY + 1 : 0) * RW + 4 + 4 * hx;
    }
    bool hcol = false; int off_x = 0, idx_x = 0, xc0 = 0, xc1 = 0;
    if (tid < 2 * LY) {
        const int rr = tid >> 1, side = tid & 1;
        hcol = true;
        xc0 = side ? x0 + 4 * LX : x0 - 1; xc1 = y0 + rr;
        off_x = WL_OFF + fa_src(xc0, g.n[0], g.per[0]) + fa_src(xc1, g.n[1], g.per[1]) * sy;
        idx_x = (rr + 1) * RW + (side ? 4 + 4 * LX : 3);
    }
    const unsigned sraw = (unsigned)__cvta_generic_to_shared(raw);
    // plane p into stage slot `slot`
    auto issue = [&](int p, int slot) {
        if (BULK) {
            if (p <= z1 + 1 && tid == 0) {
                const unsigned bar = mbar + 8u * (unsigned)slot;
                const unsigned dst = sraw + 4u * (unsigned)(slot * SP);
                const int zc_ = fa_src(p, g.n[2], g.per[2]);
                mbar_expect_tx(bar, (unsigned)(NA * PL * 4));
                tma_box3(dst, tm_r, WL_OFF + x0 - 4, y0 - 1, zc_, bar);
                if (!FIRST) tma_box3(dst + 4u * PLR, tm_e, WL_OFF + x0 - 4, y0 - 1, zc_, bar);
            }
            return;
        }
        if (p <= z1 + 1) {
            const unsigned st = sraw + 4u * (unsigned)(slot * SP);
            const int zo = fa_src(p, g.n[2], g.per[2]) * sz;
            if (own) { cp16(st + 4u * idx_own, r + (off_own + zo)); if (!FIRST) cp16(st + 4u * (PLR + idx_own), ein + (off_own + zo)); }
            if (hrow) { cp16(st + 4u * idx_h, r + (off_h + zo)); if (!FIRST) cp16(st + 4u * (PLR + idx_h), ein + (off_h + zo)); }
            if (hcol) { cp4(st + 4u * idx_x, r + (off_x + zo)); if (!FIRST) cp4(st + 4u * (PLR + idx_x), ein + (off_x + zo)); }
        }
        cp_commit();                          // one group per plane, empty past the end: the wait counts stay fixed
    };
    // ---- analytic coefficients and 1/D of this thread's cells (without the z part)
    float cxl[4], cxh[4], cyl = Lc, cyh = Lc;
    float d_in[4], d_bz[4];                   // 1/D of the own cells on a plane without / with a z boundary face
    float dh_in[4], dh_bz[4], dx_in = iDc, dx_bz = iDc;     // ... of the halo-row group and the halo-column cell
#pragma unroll
    for (int k = 0; k < 4; ++k) { cxl[k] = Lc; cxh[k] = Lc; d_in[k] = iDc; d_bz[k] = iDc; dh_in[k] = iDc; dh_bz[k] = iDc; }
    if (PLB) {
        const int byo = fa_bnd(c1, g.n[1], g.per[1]), byh = fa_bnd(hc1, g.n[1], g.per[1]);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (!g.per[0] && c0 + k == 1) cxl[k] = 0.0f;
            if (!g.per[0] && c0 + k == g.n[0]) cxh[k] = 0.0f;
            const int bo = byo + fa_bnd(c0 + k, g.n[0], g.per[0]), bh = byh + fa_bnd(hc0 + k, g.n[0], g.per[0]);
            d_in[k] = fa_pick(T, bo); d_bz[k] = fa_pick(T, bo + 1);
            dh_in[k] = fa_pick(T, bh); dh_bz[k] = fa_pick(T, bh + 1);
        }
        if (!g.per[1] && c1 == 1) cyl = 0.0f;
        if (!g.per[1] && c1 == g.n[1]) cyh = 0.0f;
        const int bx = fa_bnd(xc0, g.n[0], g.per[0]) + fa_bnd(xc1, g.n[1], g.per[1]);
        dx_in = fa_pick(T, bx); dx_bz = fa_pick(T, bx + 1);
    }
    // e' of plane p from stage slot `slot`: own group -> registers (+ shared when FULL), halo row and column -> shared
    auto form = [&](int p, int slot, float (&ep)[4], float (&rm)[4], bool full) {
        const float* st = raw + slot * SP;
        float* eb = ebuf + (p & 1) * PL;
        const bool bz = PLB && fa_bnd(p, g.n[2], g.per[2]);     // block-uniform
        if (!own) {
#pragma unroll
            for (int k = 0; k < 4; ++k) { ep[k] = 0.0f; rm[k] = 0.0f; }
        } else {
            const float4 rr = *reinterpret_cast<const float4*>(st + idx_own);
            float4 ee = make_float4(0.f, 0.f, 0.f, 0.f);
            if (!FIRST) ee = *reinterpret_cast<const float4*>(st + PLR + idx_own);
            ep[0] = fa_dir<FIRST>(ee.x, rr.x, bz ? d_bz[0] : d_in[0], beta, m); ep[1] = fa_dir<FIRST>(ee.y, rr.y, bz ? d_bz[1] : d_in[1], beta, m);
            ep[2] = fa_dir<FIRST>(ee.z, rr.z, bz ? d_bz[2] : d_in[2], beta, m); ep[3] = fa_dir<FIRST>(ee.w, rr.w, bz ? d_bz[3] : d_in[3], beta, m);
            if (FIRST) { rm[0] = rr.x - m; rm[1] = rr.y - m; rm[2] = rr.z - m; rm[3] = rr.w - m; }
        }
        if (!full) return;
        *reinterpret_cast<float4*>(eb + idx_own) = make_float4(ep[0], ep[1], ep[2], ep[3]);
        if (hrow) {
            const float4 rr = *reinterpret_cast<const float4*>(st + idx_h);
            float4 ee = make_float4(0.f, 0.f, 0.f, 0.f);
            if (!FIRST) ee = *reinterpret_cast<const float4*>(st + PLR + idx_h);
            *reinterpret_cast<float4*>(eb + idx_h) =
                make_float4(fa_dir<FIRST>(ee.x, rr.x, bz ? dh_bz[0] : dh_in[0], beta, m), fa_dir<FIRST>(ee.y, rr.y, bz ? dh_bz[1] : dh_in[1], beta, m),
                            fa_dir<FIRST>(ee.z, rr.z, bz ? dh_bz[2] : dh_in[2], beta, m), fa_dir<FIRST>(ee.w, rr.w, bz ? dh_bz[3] : dh_in[3], beta, m));
        }
        if (hcol) {
            const float rr = st[idx_x];
            const float ee = FIRST ? 0.0f : st[PLR + idx_x];
            eb[idx_x] = fa_dir<FIRST>(ee, rr, bz ? dx_bz : dx_in, beta, m);
        }
    };

    // a tile cut by a body (GEN): 1/D of plane p is loaded, at the positions the operands come from, BEFORE the wait for
    // the plane's operands, so that its latency hides behind that wait
    auto load_iD = [&](int p, bool full) {
        const int zo = fa_src(p, g.n[2], g.per[2]) * sz;
        if (own) unpack4(ld4(iD, off_own + zo), d_in);
        if (full && hrow) unpack4(ld4(iD, off_h + zo), dh_in);
        if (full && hcol) dx_in = ld1(iD, off_x + zo);
    };

    __syncthreads();                          // the previous tile's shared planes are no longer read
    // ---- prologue: planes z0-1 (own column only) in slot FA_S-1, z0 (full) in slot 0, then FA_S-1 planes ahead
    float zm[4], zc[4], zp[4], rmc[4] = { 0.f, 0.f, 0.f, 0.f }, rmp[4] = { 0.f, 0.f, 0.f, 0.f }, dummy[4];
    auto arrived = [&](int slot) {            // BULK: the plane in `slot` has landed (all threads wait on its barrier)
        mbar_wait(mbar + 8u * (unsigned)slot, (phases >> slot) & 1u);
        phases ^= 1u << slot;
    };
    issue(z0 - 1, FA_S - 1);
    issue(z0, 0);
    if (GEN) load_iD(z0 - 1, false);
    if (BULK) { arrived(FA_S - 1); arrived(0); }
    else { cp_wait<0>(); __syncthreads(); }
    form(z0 - 1, FA_S - 1, zm, dummy, false);
    if (GEN) load_iD(z0, true);
    form(z0, 0, zc, rmc, true);
    __syncthreads();                          // slot FA_S-1 is free again
#pragma unroll
    for (int d = 1; d < FA_S; ++d) issue(z0 + d, d);
    int sl = 0;                               // slot of plane z
    // ---- march
    for (int z = z0; z <= z1; ++z) {
        const int sn = sl + 1 == FA_S ? 0 : sl + 1;       // slot of plane z+1
        float lx[5] = { 0.f, 0.f, 0.f, 0.f, 0.f }, ly[4] = { 0.f, 0.f, 0.f, 0.f }, lyp[4] = { 0.f, 0.f, 0.f, 0.f };
        float lz[4] = { 0.f, 0.f, 0.f, 0.f }, lzp[4] = { 0.f, 0.f, 0.f, 0.f };
        if (GEN) {                            // 1/D of plane z+1 and the face coefficients of the own cells of plane z (L = mu0 on level 0)
            load_iD(z + 1, true);
            if (valid) {
                const int i = off_own + z * sz;
                const float4 a = ld4(L, i);
                lx[0] = a.x; lx[1] = a.y; lx[2] = a.z; lx[3] = a.w; lx[4] = ld1(L, i + 4);
                unpack4(ld4(L + g.nalloc, i), ly); unpack4(ld4(L + g.nalloc, i + sy), lyp);
                unpack4(ld4(L + 2 * g.nalloc, i), lz); unpack4(ld4(L + 2 * g.nalloc, i + sz), lzp);
            }
        }
        if (BULK) arrived(sn);
        else cp_wait<FA_S - 2>();             // plane z+1 has landed (this thread's copies) ...
        __syncthreads();                      // ... and everybody's; e'(z) in shared is complete; the slot of plane z is free
        issue(z + FA_S, sl);
        form(z + 1, sn, zp, rmp, true);
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
        float qq[4];
        if (GEN) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float ec = w[k + 1];
                float a = 0.0f;
                a += lx[k + 1] * (w[k + 2] - ec) - lx[k] * (ec - w[k]);
                a += lyp[k] * (ypv[k] - ec) - ly[k] * (ec - ymv[k]);
                a += lzp[k] * (zp[k] - ec) - lz[k] * (ec - zm[k]);
                qq[k] = a;
            }
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float ec = w[k + 1];
                float a = 0.0f;
                a += cxh[k] * (w[k + 2] - ec) - cxl[k] * (ec - w[k]);
                a += cyh * (ypv[k] - ec) - cyl * (ec - ymv[k]);
                a += czh * (zp[k] - ec) - czl * (ec - zm[k]);
                qq[k] = a;
            }
        }
        if (valid) {
            const int i = off_own + z * sz;     // own row is interior here: fa_src(c1) == c1
            *reinterpret_cast<float4*>(eout + i) = make_float4(zc[0], zc[1], zc[2], zc[3]);
            *reinterpret_cast<float4*>(q + i) = make_float4(qq[0], qq[1], qq[2], qq[3]);
            // fp32 products summed over the thread's four cells, accumulated in fp64 once per plane
            float sg = qq[0] * zc[0], sr = 0.0f;
            sg = __fmaf_rn(qq[1], zc[1], sg); sg = __fmaf_rn(qq[2], zc[2], sg); sg = __fmaf_rn(qq[3], zc[3], sg);
            acc[0] += (double)sg;
            if (FIRST) {
                sr = zc[0] * rmc[0];
                sr = __fmaf_rn(zc[1], rmc[1], sr); sr = __fmaf_rn(zc[2], rmc[2], sr); sr = __fmaf_rn(zc[3], rmc[3], sr);
                acc[1] += (double)sr;
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) { zm[k] = zc[k]; zc[k] = zp[k]; rmc[k] = rmp[k]; }
        sl = sn;
    }
    if (!BULK) cp_wait<0>();                  // drain the (empty) tail groups before the stages are reused
}

template <int FIRST, int LXL, int BULK>
__global__ void __launch_bounds__(WL_VB, WL_FA_MINB) k_pcg_A_fast(Grid g, VT vt, const int* __restrict__ plain, float Lc, float iDc,
                                                          const float* __restrict__ ein, const float* __restrict__ r,
                                                          const float* __restrict__ L, const float* __restrict__ iD,
                                                          float* __restrict__ eout, float* __restrict__ q, PcgScal* sc, RedBuf rb,
                                                          const __grid_constant__ CUtensorMap tm_r, const __grid_constant__ CUtensorMap tm_e)
{
    extern __shared__ __align__(128) float4 fa_smem4[];
    float* sm = reinterpret_cast<float*>(fa_smem4);
    if (!FIRST && !sc->live) return;          // uniform across the grid: written by an earlier kernel
    const float beta = FIRST ? 0.0f : (float)sc->beta;
    const float m = FIRST ? (sc->nlive > 0.0 ? (float)(sc->rsum / sc->nlive) : 0.0f) : 0.0f;
    constexpr int NA = FIRST ? 1 : 2;         // raw arrays per stage: r (+ e)
    constexpr int LX = 1 << LXL, LY = WL_VB >> LXL;
    constexpr int PL = (4 * LX + 8) * (LY + 2);   // floats per shared plane: rows y0-1 .. y0+LY of [3 pad][x0-1][4 LX cells][x0+4LX][3 pad]
    float* raw = sm;                          // [FA_S][NA][PL]
    constexpr int PLR = BULK ? (PL + 31) / 32 * 32 : PL;
    float* ebuf = sm + FA_S * NA * PLR;       // [2][PL]   e' of the plane being computed / the next one
    const unsigned mbar = (unsigned)__cvta_generic_to_shared(sm + FA_S * NA * PLR + 2 * PL);     // [FA_S] stage barriers (BULK)
    unsigned phases = 0;                      // parity of the next completion of each stage barrier
    if (BULK) {
        if (threadIdx.x == 0) {
#pragma unroll
            for (int k = 0; k < FA_S; ++k) mbar_init(mbar + 8u * k, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
    }
    FaTab T;
    T.t0 = 1.0f / (-6.0f * Lc); T.t1 = 1.0f / (-5.0f * Lc); T.t2 = 1.0f / (-4.0f * Lc); T.t3 = 1.0f / (-3.0f * Lc);
    double acc[2] = { 0.0, 0.0 };
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        const int mode = plain[tile];         // block-uniform
        if (mode == TM_PLI)      fa_tile<FIRST, TM_PLI, LXL, BULK>(g, vt, tile, Lc, iDc, T, beta, m, ein, r, L, iD, eout, q, raw, ebuf, acc, mbar, phases, &tm_r, &tm_e);
        else if (mode == TM_PLB) fa_tile<FIRST, TM_PLB, LXL, BULK>(g, vt, tile, Lc, iDc, T, beta, m, ein, r, L, iD, eout, q, raw, ebuf, acc, mbar, phases, &tm_r, &tm_e);
        else                     fa_tile<FIRST, TM_GEN, LXL, BULK>(g, vt, tile, Lc, iDc, T, beta, m, ein, r, L, iD, eout, q, raw, ebuf, acc, mbar, phases, &tm_r, &tm_e);
    }
    if (grid_reduce<2, OpSum>(acc, rb)) {
        if (threadIdx.x == 0) {
            const double gamma = acc[0];
            int live = 1;
            if (FIRST) {
                sc->rho = acc[1]; sc->rho0 = acc[1]; sc->beta = 0.0;
                live = fabs(acc[1]) < WL_TAU ? 0 : 1;
            }
            sc->gamma = gamma;
            if (gamma == 0.0 || !isfinite(gamma) || !live) { sc->live = 0; sc->alpha = 0.0; }
            else { sc->live = 1; sc->alpha = sc->rho / gamma; }
        }
    }
}

size_t wl_pcg_fast_smem(const VT& vt, int first, int bulk)
{
    const int LX = 1 << vt.lxl, LY = WL_VB >> vt.lxl;
    const size_t PL = (size_t)(4 * LX + 8) * (LY + 2), PLR = bulk ? (PL + 31) / 32 * 32 : PL;
    return sizeof(float) * (PLR * FA_S * (first ? 1 : 2) + 2 * PL) + 8 * FA_S + 8;      // + the stage barriers
}

// levels the shared-memory kernel takes: 3-D, whole float4 groups per row, 32-bit element offsets, 8..32 threads along x
int wl_pcg_fast_ok(const wl_sim* s, int l)
{
    const Level& lv = s->lev[l];
    return s->nd == 3 && lv.g.n[0] % 4 == 0 && lv.g.nalloc < ((int64_t)1 << 31) && lv.vt.lxl >= 3 && lv.vt.lxl <= 5;
}

// pass A on level l (every tile mode)
void wl_k_pcg_A_fast(wl_sim* s, int l, int first, const float* ein, float* eout)
{
    Level& lv = s->lev[l];
    PcgScal* sc = &s->ds->pcg[l];
    int grid = lv.vt.ntiles < s->sm_count * 4 ? lv.vt.ntiles : s->sm_count * 4;
    if (grid > WL_MAX_PARTIALS) grid = WL_MAX_PARTIALS;
    ProfScope ps_(s, WLK_PCG_MATVEC, l > 0);
#define FA_LAUNCH(F, X, B)                                                                                                          \
    do {                                                                                                                           \
        if (smem > 48 * 1024) cudaFuncSetAttribute(k_pcg_A_fast<F, X, B>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
        k_pcg_A_fast<F, X, B><<<grid, WL_VB, smem, s->st>>>(lv.g, lv.vt, lv.plain, lv.Lc, lv.iDc, ein, lv.r, lv.L, lv.iD, eout,     \
                                                            lv.q, sc, s->rb, tm_r, tm_e);                                          \
    } while (0)
    // TMA boxes where one box is all a plane needs: 32 threads along x, no wrap in x or y, tiles that fill their rows
    int bulk = s->bulk_A && lv.vt.lxl == 5 && !lv.g.per[0] && !lv.g.per[1] && lv.vt.ngx % 32 == 0;
    CUtensorMap tm_r, tm_e;
    memset(&tm_r, 0, sizeof(tm_r)); memset(&tm_e, 0, sizeof(tm_e));
    if (bulk) {
        const CUtensorMap* pr = wl_tensor_map_cached(s->tmc, lv.r, lv.g, 4 * 32 + 8, 8 + 2);
        const CUtensorMap* pe = first ? pr : wl_tensor_map_cached(s->tmc, ein, lv.g, 4 * 32 + 8, 8 + 2);
        bulk = pr && pe;
        if (bulk) { tm_r = *pr; if (!first) tm_e = *pe; }
    }
    const size_t smem = wl_pcg_fast_smem(lv.vt, first, bulk);
    switch (lv.vt.lxl) {
    case 5:
        if (bulk) { if (first) FA_LAUNCH(1, 5, 1); else FA_LAUNCH(0, 5, 1); }
        else      { if (first) FA_LAUNCH(1, 5, 0); else FA_LAUNCH(0, 5, 0); }
        break;
    case 4: if (first) FA_LAUNCH(1, 4, 0); else FA_LAUNCH(0, 4, 0); break;
    default: if (first) FA_LAUNCH(1, 3, 0); else FA_LAUNCH(0, 3, 0); break;    // wl_pcg_fast_ok() admits lxl 3..5 only
    }
#undef FA_LAUNCH
}
