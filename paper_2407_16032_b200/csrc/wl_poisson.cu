// wl_poisson.cu -- pressure projection: variable-coefficient Poisson problem solved by a
// geometric multigrid V-cycle with a Jacobi-preconditioned CG smoother (
// readings R-O, R-S, R-T of DESIGN.md).
//   (A x)_c = sum_i L[c+d_i,i](x[c+d_i]-x[c]) - L[c,i](x[c]-x[c-d_i]),  L = mu0 on level 0
// Periodic directions are handled by index wrap at load time: scalar level arrays keep no
// ghost values.  On non-periodic boundaries L = 0 on the boundary faces, so the (zero) ghost
// values never contribute.  Dot products stay on the device (PcgScal).
#include <cstdio>
#include "wl_internal.h"

// neighbour offsets of cell (c0,c1,c2) with periodic wrap: om[d] = index of c - e_d, op[d] = c + e_d
template <int ND>
__device__ __forceinline__ void nbr(const Grid& g, int c0, int c1, int c2, int64_t id, int64_t (&om)[3], int64_t (&op)[3])
{
    const int c[3] = { c0, c1, c2 };
    const int64_t st[3] = { 1, g.sy, g.sz };
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        om[d] = id - st[d];
        op[d] = id + st[d];
        if (g.per[d]) {
            if (c[d] == 1) om[d] = id + (int64_t)(g.n[d] - 1) * st[d];
            if (c[d] == g.n[d]) op[d] = id - (int64_t)(g.n[d] - 1) * st[d];
        }
    }
}

// A x at one cell.  L at the upper face of c in direction d is L_d[c + e_d] (wrapped).
template <int ND>
__device__ __forceinline__ float apply_A(const Grid& g, const float* __restrict__ L, const float* __restrict__ x,
                                         int64_t id, const int64_t (&om)[3], const int64_t (&op)[3])
{
    const float xc = x[id];
    float acc = 0.0f;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        const float* Ld = L + d * g.nalloc;
        acc += Ld[op[d]] * (x[op[d]] - xc) - Ld[id] * (xc - x[om[d]]);
    }
    return acc;
}

// ---- Poisson diagonal: D = -sum_i (L[c,i] + L[c+d_i,i]); iD = 1/D if |D| > 2n*1e-6 else 0
// (R-O: cells buried in the body, or within ~1e-2 eps of being so, decouple)
template <int ND>
__global__ void __launch_bounds__(512) k_diag(Grid g, Tiling T, const float* __restrict__ L, float* __restrict__ iD)
{
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2), om[3], op[3];
        nbr<ND>(g, c0, c1, c2, id, om, op);
        float D = 0.0f;
#pragma unroll
        for (int d = 0; d < ND; ++d) D -= L[d * g.nalloc + id] + L[d * g.nalloc + op[d]];
        iD[id] = fabsf(D) > 2.0f * ND * 1e-6f ? 1.0f / D : 0.0f;
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

// ---- project!, first half (R-K): pscale = w dt; x = pscale p; r = div u - A x.
template <int ND>
__global__ void __launch_bounds__(512) k_residual(Grid g, Tiling T, const float* __restrict__ u, const float* __restrict__ L,
                                                  const float* __restrict__ p, float* __restrict__ x, float* __restrict__ r,
                                                  DevScal* ds, float w)
{
    const float sc = w * ds->dt;
    if (blockIdx.x == 0 && threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) ds->pscale = sc;
    const int64_t st[3] = { 1, g.sy, g.sz };
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2), om[3], op[3];
        nbr<ND>(g, c0, c1, c2, id, om, op);
        float div = 0.0f;
#pragma unroll
        for (int d = 0; d < ND; ++d) div += u[d * g.nalloc + id + st[d]] - u[d * g.nalloc + id];   // u ghosts are BC-filled
        const float xc = sc * p[id];
        float acc = 0.0f;
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            const float* Ld = L + d * g.nalloc;
            acc += Ld[op[d]] * (sc * p[op[d]] - xc) - Ld[id] * (xc - sc * p[om[d]]);
        }
        x[id] = xc;
        r[id] = div - acc;
    }
}

// ---- project!, second half (P:88 kernel): u[c,i] -= L[c,i] (x[c] - x[c-d_i]); p = x / pscale
template <int ND>
__global__ void __launch_bounds__(512) k_apply_gradient(Grid g, Tiling T, float* __restrict__ u, const float* __restrict__ L,
                                                        const float* __restrict__ x, float* __restrict__ p, const DevScal* __restrict__ ds)
{
    const float isc = 1.0f / ds->pscale;
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2), om[3], op[3];
        nbr<ND>(g, c0, c1, c2, id, om, op);
        const float xc = x[id];
#pragma unroll
        for (int d = 0; d < ND; ++d) u[d * g.nalloc + id] -= L[d * g.nalloc + id] * (xc - x[om[d]]);
        p[id] = xc * isc;
    }
}

// ---- residual restriction: r_c[C] = sum of the 2^n children; x_c = 0 (R-S)
template <int ND>
__global__ void __launch_bounds__(512) k_restrict_r(Grid gf, Grid gc, Tiling T, const float* __restrict__ rf, float* __restrict__ rc, float* __restrict__ xc)
{
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int C0, C1, C2;
        if (!tile_cell(T, tile, C0, C1, C2)) continue;
        float sum = 0.0f;
        const int n2 = ND == 3 ? 2 : 1;
        for (int a2 = 0; a2 < n2; ++a2)
            for (int a1 = 0; a1 < 2; ++a1) {
                int64_t b = gidx(gf, 2 * C0 - 1, 2 * C1 - 1 + a1, ND == 3 ? 2 * C2 - 1 + a2 : 0);
                sum += rf[b];
                sum += rf[b + 1];
            }
        int64_t idc = gidx(gc, C0, C1, C2);
        rc[idc] = sum;
        xc[idc] = 0.0f;
    }
}

// ---- prolongation + increment: e = P x_c (piecewise constant); x_f += e; r_f -= A_f e (R-S)
template <int ND>
__global__ void __launch_bounds__(512) k_prolong(Grid gf, Grid gc, Tiling T, const float* __restrict__ L, const float* __restrict__ xc,
                                                 float* __restrict__ xf, float* __restrict__ rf)
{
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c[3];
        if (!tile_cell(T, tile, c[0], c[1], c[2])) continue;
        int64_t id = gidx(gf, c[0], c[1], c[2]), om[3], op[3];
        nbr<ND>(gf, c[0], c[1], c[2], id, om, op);
        const float ec = xc[gidx(gc, (c[0] + 1) >> 1, (c[1] + 1) >> 1, ND == 3 ? (c[2] + 1) >> 1 : 0)];
        float acc = 0.0f;
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            // parents of the two neighbours in direction d (wrapped); outside a non-periodic
            // boundary the face coefficient is zero, any finite value does
            int cm[3] = { c[0], c[1], c[2] }, cp[3] = { c[0], c[1], c[2] };
            cm[d] = wrapc(c[d] - 1, gf.n[d], gf.per[d]);
            cp[d] = wrapc(c[d] + 1, gf.n[d], gf.per[d]);
            float em = cm[d] >= 1 ? xc[gidx(gc, (cm[0] + 1) >> 1, (cm[1] + 1) >> 1, ND == 3 ? (cm[2] + 1) >> 1 : 0)] : 0.0f;
            float ep = cp[d] <= gf.n[d] ? xc[gidx(gc, (cp[0] + 1) >> 1, (cp[1] + 1) >> 1, ND == 3 ? (cp[2] + 1) >> 1 : 0)] : 0.0f;
            const float* Ld = L + d * gf.nalloc;
            acc += Ld[op[d]] * (ep - ec) - Ld[id] * (ec - em);
        }
        xf[id] += ec;
        rf[id] -= acc;
    }
}

// ---- Jacobi-preconditioned CG smoother (R-S, R-T), restarted at every call:
//   z = e = iD r; rho = r.z; if |rho| < tau return
//   loop k = 1..it: q = A e; gamma = q.e; alpha = rho/gamma; x += alpha e; r -= alpha q;
//                   if k == it break; z = iD r; rho' = r.z; if |rho'| < tau or < theta |rho0| break;
//                   beta = rho'/rho; e = beta e + z; rho = rho'
template <int ND>
__global__ void __launch_bounds__(512) k_pcg_init(Grid g, Tiling T, const float* __restrict__ r, const float* __restrict__ iD,
                                                  float* __restrict__ e, PcgScal* sc, RedBuf rb)
{
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        float rr = r[id], z = iD[id] * rr;
        e[id] = z;
        v[0] += (double)z * (double)rr;
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) {
            sc->rho = v[0];
            sc->rho0 = v[0];
            sc->live = fabs(v[0]) < WL_TAU ? 0 : 1;
            sc->alpha = 0.0; sc->beta = 0.0; sc->gamma = 0.0;
        }
    }
}

template <int ND>
__global__ void __launch_bounds__(512) k_pcg_matvec(Grid g, Tiling T, const float* __restrict__ L, const float* __restrict__ e,
                                                    float* __restrict__ q, PcgScal* sc, RedBuf rb)
{
    if (!sc->live) return;          // uniform across the grid: written by an earlier kernel
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2), om[3], op[3];
        nbr<ND>(g, c0, c1, c2, id, om, op);
        float a = apply_A<ND>(g, L, e, id, om, op);
        q[id] = a;
        v[0] += (double)a * (double)e[id];
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) {
            double gamma = v[0];
            sc->gamma = gamma;
            if (gamma == 0.0 || !isfinite(gamma)) { sc->live = 0; sc->alpha = 0.0; }
            else sc->alpha = sc->rho / gamma;
        }
    }
}

// x += alpha e; r -= alpha q; unless last: z = iD r (stored in q), rho' = r.z -> beta
template <int ND>
__global__ void __launch_bounds__(512) k_pcg_update(Grid g, Tiling T, float* __restrict__ x, float* __restrict__ r, const float* __restrict__ e,
                                                    float* __restrict__ q, const float* __restrict__ iD, PcgScal* sc, RedBuf rb, int last)
{
    if (!sc->live) return;
    const float alpha = (float)sc->alpha;
    double v[1] = { 0.0 };
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        x[id] += alpha * e[id];
        float rr = r[id] - alpha * q[id];
        r[id] = rr;
        if (!last) {
            float z = iD[id] * rr;
            q[id] = z;
            v[0] += (double)z * (double)rr;
        }
    }
    if (last) return;
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) {
            double rho2 = v[0];
            if (fabs(rho2) < WL_TAU || fabs(rho2) < WL_THETA * fabs(sc->rho0)) sc->live = 0;
            else { sc->beta = rho2 / sc->rho; sc->rho = rho2; }
        }
    }
}

// e = beta e + z
template <int ND>
__global__ void __launch_bounds__(512) k_pcg_dir(Grid g, Tiling T, float* __restrict__ e, const float* __restrict__ z, const PcgScal* __restrict__ sc)
{
    if (!sc->live) return;
    const float beta = (float)sc->beta;
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        e[id] = beta * e[id] + z[id];
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
        Tiling T = wl_tiles_interior(s, lv.g);
        DISPATCH(s, WLK_POISSON_UPDATE, l > 0, k_diag, T, lv.g, T, lv.L, lv.iD);
    }
}

void wl_k_residual(wl_sim* s, const float* u, float w)
{
    Level& lv = s->lev[0];
    Tiling T = wl_tiles_interior(s, lv.g);
    DISPATCH(s, WLK_RESIDUAL, 0, k_residual, T, lv.g, T, u, lv.L, s->p, lv.x, lv.r, s->ds, w);
}

void wl_k_apply_gradient(wl_sim* s, float* u)
{
    Level& lv = s->lev[0];
    Tiling T = wl_tiles_interior(s, lv.g);
    DISPATCH(s, WLK_GRADIENT, 0, k_apply_gradient, T, lv.g, T, u, lv.L, lv.x, s->p, s->ds);
}

void wl_k_restrict(wl_sim* s, int l)
{
    Level &lf = s->lev[l], &lc = s->lev[l + 1];
    Tiling T = wl_tiles_interior(s, lc.g);
    DISPATCH(s, WLK_RESTRICT, l > 0, k_restrict_r, T, lf.g, lc.g, T, lf.r, lc.r, lc.x);
}

void wl_k_prolong(wl_sim* s, int l)
{
    Level &lf = s->lev[l], &lc = s->lev[l + 1];
    Tiling T = wl_tiles_interior(s, lf.g);
    DISPATCH(s, WLK_PROLONG, l > 0, k_prolong, T, lf.g, lc.g, T, lf.L, lc.x, lf.x, lf.r);
}

void wl_k_smooth(wl_sim* s, int l, int iters)
{
    Level& lv = s->lev[l];
    Tiling T = wl_tiles_interior(s, lv.g);
    PcgScal* sc = &s->ds->pcg[l];
    DISPATCH(s, WLK_PCG_INIT, l > 0, k_pcg_init, T, lv.g, T, lv.r, lv.iD, lv.e, sc, s->rb);
    for (int k = 1; k <= iters; ++k) {
        DISPATCH(s, WLK_PCG_MATVEC, l > 0, k_pcg_matvec, T, lv.g, T, lv.L, lv.e, lv.q, sc, s->rb);
        DISPATCH(s, WLK_PCG_UPDATE, l > 0, k_pcg_update, T, lv.g, T, lv.x, lv.r, lv.e, lv.q, lv.iD, sc, s->rb, k == iters ? 1 : 0);
        if (k == iters) break;
        DISPATCH(s, WLK_PCG_DIR, l > 0, k_pcg_dir, T, lv.g, T, lv.e, lv.q, sc);
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
