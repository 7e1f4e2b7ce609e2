// wl_flow.cu -- flow-side kernels of libwl: body measurement, boundary conditions, convective
// exit, CFL reduction, pressure force, initial conditions, pack/unpack of user buffers.
// Citations "P:<line>" are /root/reference/PAPER.md; "R-<x>" are the readings of DESIGN.md s.3.
#include <cstdio>
#include <cstring>
#include "wl_internal.h"

// ------------------------------------------------------------------ time / body state
// One thread.  Sets the running dt (host value, or the device-resident CFL result) and the time at which the body is
// placed (host value, or t_step + dt: reading R-R), then the translation map, sinusoidal in every direction,
//     c_d(t) = c0_d + amp_d sin(2 pi f_d t + phase_d),  V = dc/dt
// Modes: see wl_internal.h.  The simulation time t_step moves only with wl_step (t_mode 2 and 0), so a wl_measure or
// wl_pressure_force at some other time cannot shift the trajectory of a device-resident run.
struct BodyAll { int n; wl_body part[WLB_MAXPART]; };     // every primitive's map parameters (kernel argument)

__device__ __forceinline__ void body_place(const wl_body& b, double t, PartState& q)
{
    const double two_pi = 6.283185307179586476925286766559;
    const double phs = two_pi * (double)b.scale_freq * t + (double)b.scale_phase;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        q.c[k] = (double)b.centre[k];
        q.cdot[k] = 0.0;
        if (b.motion == WL_MOTION_SIN) {
            const double ph = two_pi * (double)b.freq[k] * t + (double)b.phase[k];
            q.c[k] += (double)b.amp[k] * sin(ph);
            q.cdot[k] = (double)b.amp[k] * two_pi * (double)b.freq[k] * cos(ph);
        }
        q.s[k] = 1.0 + (double)b.scale_amp[k] * cos(phs);
        q.sdot_s[k] = -(double)b.scale_amp[k] * two_pi * (double)b.scale_freq * sin(phs) / q.s[k];
    }
}

__global__ void k_set_time(DevScal* ds, BodyAll B, double t_host, float dt_host, int t_mode, int dt_mode)
{
    if (dt_mode == 1) ds->dt = dt_host; else if (dt_mode == 0) ds->dt = ds->dt_next;
    double t = ds->t;
    if (t_mode == 2) { t = t_host; ds->t_step = t; }
    else if (t_mode == 1) t = t_host;
    else if (t_mode == 0) { t = ds->t_step + (double)ds->dt; ds->t_step = t; }
    ds->t = t;
    for (int e = 0; e < B.n; ++e) body_place(B.part[e], t, ds->part[e]);
    for (int k = 0; k < 3; ++k) ds->vel[k] = B.n > 0 ? (float)ds->part[0].cdot[k] : 0.0f;     // one rigid translation: V is uniform
}

// the body for the pressure-force integral: at the host time t, or (t = NaN) where measure! last placed it
__global__ void k_force_time(DevScal* ds, BodyAll B, double t_host)
{
    for (int e = 0; e < B.n; ++e) {
        if (t_host == t_host) body_place(B.part[e], t_host, ds->part_f[e]);
        else ds->part_f[e] = ds->part[e];
    }
}

// ------------------------------------------------------------------ measure!
// One thread per padded cell; for each face (c,i), x_f = x_c(c) - e_i/2:
//   mu0[c,i] = mu0(d), mu1[c,i,j] = mu1(d) n_j                       (R-B, R-D, R-E)
// Periodic ghosts are evaluated at the wrapped position; on non-periodic boundaries mu0 = 0 on
// the two boundary-normal faces c_i = 1 and c_i = N_i+1 (R-O: homogeneous-Neumann Poisson
// problem).  V is a uniform vector for the translation maps supported and lives in DevScal.
template <int ND>
__global__ void __launch_bounds__(512) k_measure(Grid g, Tiling T, BodyP b, const DevScal* __restrict__ ds,
                                                 float* __restrict__ mu0, float* __restrict__ mu1, float* __restrict__ Vf,
                                                 DevScal* dsw, long long* __restrict__ band, int band_cap)
{
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c[3];
        if (!tile_cell(T, tile, c[0], c[1], c[2])) continue;
        int64_t id = gidx(g, c[0], c[1], c[2]);
        float xc[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) xc[k] = k < ND ? (float)wrapc(c[k], g.n[k], g.per[k]) - 0.5f : 0.0f;
        // A cell whose CENTRE is far out in the fluid has all its faces (half a cell away) outside the band: mu0 = 1, mu1 = 0, and V,
        // which enters only through (1 - mu0) and mu1, is not needed (k_measure_wallV supplies it on the forced boundary faces).  One fp32
        // evaluation instead of three; the margin of 2.5 cells covers the half cell and the first-order distance of a non-rigid map.
        if (b.n > 0) {
            double xd[3];
            float nf[3], vf[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) xd[k] = (double)xc[k];
            if (body_eval<ND, float>(b, ds->part, xd, nf, vf) > b.eps + 2.5f) {
#pragma unroll
                for (int i = 0; i < ND; ++i) {
                    mu0[i * g.nalloc + id] = (!g.per[i] && (c[i] == 1 || c[i] == g.n[i] + 1)) ? 0.0f : 1.0f;
#pragma unroll
                    for (int j = 0; j < ND; ++j) mu1[(i * ND + j) * g.nalloc + id] = 0.0f;
                }
                continue;
            }
        }
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            float m0 = 1.0f, m1 = 0.0f, nrm[3] = { 0.f, 0.f, 0.f }, vel[3] = { 0.f, 0.f, 0.f };
            if (b.n > 0) {
                double xf[3], nd[3];
#pragma unroll
                for (int k = 0; k < 3; ++k) xf[k] = k < ND ? (double)xc[k] - (k == i ? 0.5 : 0.0) : 0.0;
                // far from the surface (most faces) fp32 decides: further than eps, mu0 is exactly 0 or 1 and mu1 exactly 0 whatever the
                // last digits of d (its fp32 error is ~1e-4 of a cell: the margin of one cell is ample); only the band pays for fp64
                float nf[3];
                float d = body_eval<ND, float>(b, ds->part, xf, nf, vel);
                if (fabsf(d) <= b.eps + 1.0f) {
                    d = (float)body_eval<ND, double>(b, ds->part, xf, nd, vel);
#pragma unroll
                    for (int k = 0; k < 3; ++k) nrm[k] = (float)nd[k];
                }
                m0 = bdim_mu0(d, b.eps);
                m1 = bdim_mu1(d, b.eps);
            }
            if (!g.per[i] && (c[i] == 1 || c[i] == g.n[i] + 1)) m0 = 0.0f;
            mu0[i * g.nalloc + id] = m0;
            if (Vf) Vf[i * g.nalloc + id] = vel[i];
            bool any = false;
#pragma unroll
            for (int j = 0; j < ND; ++j) {
                const float v = m1 * nrm[j];
                mu1[(i * ND + j) * g.nalloc + id] = v;
                any = any || v != 0.0f;
            }
            // the band list of conv_diff!/BDIM!: interior faces whose mu1 is non-zero (entry order is
            // irrelevant: every entry is processed independently)
            bool inner = true;
#pragma unroll
            for (int k = 0; k < ND; ++k) inner = inner && c[k] >= 1 && c[k] <= g.n[k];
            if (any && inner) {
                // one third of the list per component: the band kernel's warps then work on one component each
                const int cap3 = band_cap / 3, slot = atomicAdd(&dsw->band_count[i], 1);
                if (slot < cap3) band[(int64_t)i * cap3 + slot] = ((long long)id << 2) | i;
            }
        }
    }
}

// General bodies (V is a per-face field): the boundary-normal faces c_i in {1, N_i + 1} of a non-periodic direction carry mu0 = 0
// (R-O), so BDIM! puts V there until BC! overwrites it; after the first measure! only the box the body can reach is re-measured, and
// this kernel keeps V_i on those planes current (V of a non-rigid or spinning map changes everywhere in time).
template <int ND>
__global__ void __launch_bounds__(256) k_measure_wallV(Grid g, BodyP b, const DevScal* __restrict__ ds, float* __restrict__ Vf)
{
    int64_t A[3];
    A[0] = (int64_t)g.S[1] * g.S[2]; A[1] = (int64_t)g.S[0] * g.S[2]; A[2] = (int64_t)g.S[0] * g.S[1];
    int64_t total = 0;
    for (int j = 0; j < ND; ++j) total += g.per[j] ? 0 : 2 * A[j];
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        int64_t rem = t;
        int j = 0;
        for (;; ++j) {
            const int64_t cnt = g.per[j] ? 0 : 2 * A[j];
            if (rem < cnt) break;
            rem -= cnt;
        }
        const int plane = (int)(rem / A[j]);
        const int64_t ab = rem % A[j];
        const int d0 = j == 0 ? 1 : 0, d1 = j == 2 ? 1 : 2;
        int c[3] = { 0, 0, 0 };
        c[d0] = (int)(ab % g.S[d0]);
        c[d1] = (int)(ab / g.S[d0]);
        if (ND == 2) c[2] = 0;
        c[j] = plane == 0 ? 1 : g.n[j] + 1;
        double xf[3], nd[3];
        float vel[3] = { 0.f, 0.f, 0.f };
#pragma unroll
        for (int k = 0; k < 3; ++k) xf[k] = k < ND ? (double)((float)wrapc(c[k], g.n[k], g.per[k]) - 0.5f) - (k == j ? 0.5 : 0.0) : 0.0;
        body_eval<ND, double>(b, ds->part, xf, nd, vel);
        Vf[j * g.nalloc + gidx(g, c[0], c[1], c[2])] = vel[j];
    }
}

// ------------------------------------------------------------------ BC! (R-M)
// The rule is stated direction by direction (x, then y, then z, each over the whole padded
// range of the others): periodic -> ghost := wrapped interior; otherwise the normal component
// is U_j on c_j in {0, 1, N_j+1} (the upper one is left alone on the convective exit) and the
// tangential ghosts copy the adjacent interior value (slip).  Composing the three passes, the
// final value of any shell cell is found by walking the directions from the last to the first
// and redirecting the coordinate to its source; sources are never written by this kernel.
template <int ND>
__device__ __forceinline__ float bc_resolve(const FlowP& P, const float* u, int i, const int (&c)[3], bool& self)
{
    int cc[3] = { c[0], c[1], c[2] };
#pragma unroll
    for (int j = ND - 1; j >= 0; --j) {
        const int N = P.g.n[j];
        if (P.g.per[j]) {
            if (cc[j] == 0) cc[j] = N; else if (cc[j] == N + 1) cc[j] = 1;
        } else if (i == j) {
            if (cc[j] <= 1 || (cc[j] == N + 1 && !(P.exit_bc && j == 0))) { self = false; return P.U[j]; }
        } else {
            if (cc[j] == 0) cc[j] = 1; else if (cc[j] == N + 1) cc[j] = N;
        }
    }
    self = (cc[0] == c[0] && cc[1] == c[1] && cc[2] == c[2]);
    return u[i * P.g.nalloc + gidx(P.g, cc[0], cc[1], cc[2])];
}

template <int ND>
__global__ void k_bc(FlowP P, float* u)
{
    const Grid& g = P.g;
    int64_t A[3];
    A[0] = (int64_t)g.S[1] * g.S[2]; A[1] = (int64_t)g.S[0] * g.S[2]; A[2] = (int64_t)g.S[0] * g.S[1];
    int64_t total = 0;
    for (int j = 0; j < ND; ++j) total += 3 * A[j];
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        int64_t rem = t;
        int j = 0;
        while (rem >= 3 * A[j]) { rem -= 3 * A[j]; ++j; }
        int plane = (int)(rem / A[j]);
        int64_t ab = rem % A[j];
        int c[3] = { 0, 0, 0 };
        int d0 = j == 0 ? 1 : 0;                 // fastest of the two in-plane directions
        int d1 = j == 2 ? 1 : 2;
        c[d0] = (int)(ab % g.S[d0]);
        c[d1] = (int)(ab / g.S[d0]);
        if (ND == 2) c[2] = 0;
        c[j] = plane == 0 ? 0 : (plane == 1 ? 1 : g.n[j] + 1);
        if (plane == 1 && g.per[j]) continue;
        int64_t id = gidx(g, c[0], c[1], c[2]);
#pragma unroll
        for (int i = 0; i < ND; ++i) {
            if (plane == 1 && i != j) continue;
            bool self;
            float v = bc_resolve<ND>(P, u, i, c, self);
            if (!self) u[i * g.nalloc + id] = v;
        }
    }
}

// ------------------------------------------------------------------ exitBC! (R-N)
// Exit plane c_x = N_x+1: u_x <- u0_x - U_x dt (u0_x[c] - u0_x[c - d_x]); then every value is
// shifted by (mean - U_x) so that outflow = nominal inflow.
template <int ND>
__global__ void __launch_bounds__(256) k_exit_a(FlowP P, float* u, const float* __restrict__ u0, DevScal* ds, RedBuf rb)
{
    const Grid& g = P.g;
    const int n1 = g.n[1], n2 = ND == 3 ? g.n[2] : 1;
    const int cnt = n1 * n2;
    const float dt = ds->dt;
    double v[1] = { 0.0 };
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < cnt; t += gridDim.x * blockDim.x) {
        int c1 = 1 + t % n1, c2 = ND == 3 ? 1 + t / n1 : 0;
        int64_t id = gidx(g, g.n[0] + 1, c1, c2);
        float a = u0[id], b = u0[id - 1];
        float val = a - P.U[0] * dt * (a - b);
        u[id] = val;
        v[0] += (double)val;
    }
    if (grid_reduce<1, OpSum>(v, rb)) {
        if (threadIdx.x == 0) ds->exit_corr = (float)(v[0] / (double)cnt - (double)P.U[0]);
    }
}
template <int ND>
__global__ void k_exit_b(FlowP P, float* u, const DevScal* __restrict__ ds)
{
    const Grid& g = P.g;
    const int n1 = g.n[1], n2 = ND == 3 ? g.n[2] : 1;
    const int cnt = n1 * n2;
    const float corr = ds->exit_corr;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < cnt; t += gridDim.x * blockDim.x) {
        int c1 = 1 + t % n1, c2 = ND == 3 ? 1 + t / n1 : 0;
        u[gidx(g, g.n[0] + 1, c1, c2)] -= corr;
    }
}

// ------------------------------------------------------------------ CFL! (R-U)
// dt = min(dt_max, cfl_c / (max_c sum_i [max(0,u_i[c+d_i]) + max(0,-u_i[c])] + cfl_cnu nu))
// One thread per four consecutive x cells (float4 loads), marching along z with the lower z face in registers.
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_cfl(Grid g, VT vt, const float* __restrict__ u, DevScal* ds, RedBuf rb,
                                               float nu, float cfl_c, float cfl_cnu, float dt_max)
{
    double v[2] = { 0.0, 0.0 };
    float amax = 0.0f;
    bool bad = false;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
        const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + p.c0;
        float wl[4] = { 0.f, 0.f, 0.f, 0.f };
        if (ND == 3) unpack4(ld4(u + 2 * g.nalloc, rc + (int64_t)p.z0 * g.sz), wl);
        for (int z = p.z0; z <= p.z1; ++z) {
            const int64_t i = rc + (int64_t)z * g.sz;
            float ux[4], vy[4], vyp[4], wu[4] = { 0.f, 0.f, 0.f, 0.f };
            unpack4(ld4(u, i), ux);
            const float ux4 = ld1(u, i + 4);                 // ghosts are BC-filled: plain +1 neighbours
            unpack4(ld4(u + g.nalloc, i), vy);
            unpack4(ld4(u + g.nalloc, i + g.sy), vyp);
            if (ND == 3) unpack4(ld4(u + 2 * g.nalloc, i + g.sz), wu);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float up = k < 3 ? ux[k + 1] : ux4;
                float a = fmaxf(up, 0.0f) + fmaxf(-ux[k], 0.0f);
                a += fmaxf(vyp[k], 0.0f) + fmaxf(-vy[k], 0.0f);
                if (ND == 3) a += fmaxf(wu[k], 0.0f) + fmaxf(-wl[k], 0.0f);
                if (k < p.nv) {
                    amax = fmaxf(amax, a);
                    bad = bad || !isfinite(up) || !isfinite(ux[k]) || !isfinite(vy[k]) || !isfinite(vyp[k]) || !isfinite(wu[k]) || !isfinite(wl[k]);
                }
                wl[k] = wu[k];
            }
        }
    }
    v[0] = (double)amax;
    v[1] = bad ? 1.0 : 0.0;
    if (grid_reduce<2, OpMax>(v, rb)) {
        if (threadIdx.x == 0) {
            float m = (float)v[0];
            float dt = cfl_c / (m + cfl_cnu * nu);
            ds->dt_next = dt < dt_max ? dt : dt_max;
            ds->cfl_max = v[0];
            ds->nan_flag = v[1] > 0.5 ? 1 : 0;
        }
    }
}

// ------------------------------------------------------------------ pressure force (R-Z)
// F = - sum_{c interior} p[c] n(x_c) K^{1}(d(x_c)), one-cell-wide surface delta at cell centres.
template <int ND>
__global__ void __launch_bounds__(512) k_force(Grid g, Tiling T, BodyP b, const float* __restrict__ p, DevScal* ds, RedBuf rb)
{
    double v[3] = { 0.0, 0.0, 0.0 };
    if (b.n > 0) {
        for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
            int c[3];
            if (!tile_cell(T, tile, c[0], c[1], c[2])) continue;
            double xc[3];
            float nrm[3], vel[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) xc[k] = k < ND ? (double)c[k] - 0.5 : 0.0;
            float d = body_eval<ND, float>(b, ds->part_f, xc, nrm, vel);
            float kk = bdim_K(d, 1.0f);
            if (kk == 0.0f) continue;
            float pk = p[gidx(g, c[0], c[1], c[2])] * kk;
            v[0] -= (double)(pk * nrm[0]); v[1] -= (double)(pk * nrm[1]); v[2] -= (double)(pk * nrm[2]);
        }
    }
    if (grid_reduce<3, OpSum>(v, rb)) {
        if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) {
            ds->force[0] = v[0]; ds->force[1] = v[1]; ds->force[2] = v[2];
        }
    }
}

// ------------------------------------------------------------------ kinetic energy and enstrophy (Fig. 4; R-E2)
//   KE = 1/2 sum_c sum_i u_i[c]^2 ;  Z = 1/2 sum_c |w[c]|^2,  w_k[c] = (u_j[c] - u_j[c-d_i]) - (u_i[c] - u_i[c-d_j]), (i,j,k) cyclic:
// the circulation around the cell edge along k through the lower corner of cell c.  One thread per four x cells, marching
// along z with the plane below in registers; ghosts are BC-filled, so the -1 neighbours are plain loads.  fp64 partials,
// fixed tree.
template <int ND>
__global__ void __launch_bounds__(WL_VB) k_energy(Grid g, VT vt, const float* __restrict__ u, DevScal* ds, RedBuf rb)
{
    double v[2] = { 0.0, 0.0 };
    const float* ux = u; const float* uy = u + g.nalloc; const float* uz = u + 2 * g.nalloc;
    for (int tile = blockIdx.x; tile < vt.ntiles; tile += gridDim.x) {
        VPos p = vt_pos(g, vt, tile);
        if (p.nv == 0) continue;
        const int64_t rc = (int64_t)WL_OFF + (int64_t)p.c1 * g.sy + p.c0;
        float xl[4] = { 0.f, 0.f, 0.f, 0.f }, yl[4] = { 0.f, 0.f, 0.f, 0.f };      // u_x, u_y of the plane below
        if (ND == 3) { unpack4(ld4(ux, rc + (int64_t)(p.z0 - 1) * g.sz), xl); unpack4(ld4(uy, rc + (int64_t)(p.z0 - 1) * g.sz), yl); }
        for (int z = p.z0; z <= p.z1; ++z) {
            const int64_t i = rc + (int64_t)z * g.sz;
            float a[4], b[4], c[4] = { 0.f, 0.f, 0.f, 0.f }, am[4], cm[4] = { 0.f, 0.f, 0.f, 0.f };
            unpack4(ld4(ux, i), a); unpack4(ld4(uy, i), b);
            unpack4(ld4(ux, i - g.sy), am);                      // u_x one row down
            const float bl = ld1(uy, i - 1);                     // u_y one cell to the left of the group
            float cl = 0.f;
            if (ND == 3) { unpack4(ld4(uz, i), c); unpack4(ld4(uz, i - g.sy), cm); cl = ld1(uz, i - 1); }
            float ke = 0.f, en = 0.f;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (k >= p.nv) break;
                ke += a[k] * a[k] + b[k] * b[k] + c[k] * c[k];
                const float wz = (b[k] - (k == 0 ? bl : b[k - 1])) - (a[k] - am[k]);
                en += wz * wz;
                if (ND == 3) {
                    const float wx = (c[k] - cm[k]) - (b[k] - yl[k]);
                    const float wy = (a[k] - xl[k]) - (c[k] - (k == 0 ? cl : c[k - 1]));
                    en += wx * wx + wy * wy;
                }
            }
            v[0] += 0.5 * (double)ke; v[1] += 0.5 * (double)en;
#pragma unroll
            for (int k = 0; k < 4; ++k) { xl[k] = a[k]; yl[k] = b[k]; }
        }
    }
    if (grid_reduce<2, OpSum>(v, rb)) {
        if (threadIdx.x == 0) { ds->energy[0] = v[0]; ds->energy[1] = v[1]; }
    }
}

// ------------------------------------------------------------------ initial conditions
// Taylor-Green vortex (Eq. 3-5; R-W), staggered sampling, whole padded array.  One period per periodic
// direction; HALF a period in a non-periodic one, whose slip walls (U = 0) are then symmetry planes of the vortex: the
// half-domain of P:118.
template <int ND>
__global__ void __launch_bounds__(512) k_init_tgv(Grid g, Tiling T, float* u, float* p, int sign)
{
    const double two_pi = 6.283185307179586476925286766559;
    const double k0 = (g.per[0] ? 1.0 : 0.5) * two_pi / g.n[0], k1 = (g.per[1] ? 1.0 : 0.5) * two_pi / g.n[1];
    const double k2 = ND == 3 ? (g.per[2] ? 1.0 : 0.5) * two_pi / g.n[2] : 0.0;
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        double xc = c0 - 0.5, yc = c1 - 0.5, zc = ND == 3 ? c2 - 0.5 : 0.0;
        double cz = ND == 3 ? cos(k2 * zc) : 1.0;
        u[id] = (float)(sign * sin(k0 * (xc - 0.5)) * cos(k1 * yc) * cz);
        u[g.nalloc + id] = (float)(-sign * cos(k0 * xc) * sin(k1 * (yc - 0.5)) * cz);
        if (ND == 3) u[2 * g.nalloc + id] = 0.0f;
        p[id] = 0.0f;
    }
}

__global__ void k_fill(float* a, int64_t n, float v)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) a[i] = v;
}

// user buffer (the box T.o .. T.o+T.e of the padded array, dense) <-> padded array
template <int ND>
__global__ void __launch_bounds__(512) k_pack(Grid g, Tiling T, const float* __restrict__ padded, float* __restrict__ dense, int ncomp, float scale)
{
    const int64_t nint = (int64_t)T.e[0] * T.e[1] * T.e[2];
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        int64_t k = (c0 - T.o[0]) + (int64_t)T.e[0] * ((c1 - T.o[1]) + (int64_t)T.e[1] * (c2 - T.o[2]));
        for (int m = 0; m < ncomp; ++m) dense[m * nint + k] = scale * padded[m * g.nalloc + id];
    }
}
template <int ND>
__global__ void __launch_bounds__(512) k_unpack(Grid g, Tiling T, const float* __restrict__ dense, float* __restrict__ padded, int ncomp)
{
    const int64_t nint = (int64_t)T.e[0] * T.e[1] * T.e[2];
    for (int tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        int c0, c1, c2;
        if (!tile_cell(T, tile, c0, c1, c2)) continue;
        int64_t id = gidx(g, c0, c1, c2);
        int64_t k = (c0 - T.o[0]) + (int64_t)T.e[0] * ((c1 - T.o[1]) + (int64_t)T.e[1] * (c2 - T.o[2]));
        for (int m = 0; m < ncomp; ++m) padded[m * g.nalloc + id] = dense[m * nint + k];
    }
}

// ================================================================== host launchers

static BodyAll body_all(const wl_sim* s)
{
    BodyAll B;
    memset(&B, 0, sizeof(B));
    if (s->cfg.body.kind == WL_BODY_NONE) return B;
    B.n = 1 + s->cfg.nextra;
    B.part[0] = s->cfg.body;
    for (int e = 0; e < s->cfg.nextra; ++e) B.part[1 + e] = s->cfg.extra[e];
    return B;
}

void wl_k_set_time(wl_sim* s, double t, float dt, int t_mode, int dt_mode)
{
    ProfScope ps(s, WLK_SET_TIME);
    k_set_time<<<1, 1, 0, s->st>>>(s->ds, body_all(s), t, dt, t_mode, dt_mode);
}

// The box of padded cells the body can reach, grown by `margin` cells: the supported motion is a sinusoidal translation of
// known amplitude, so the box is known on the host although t is device-resident.  interior: clip to the interior cells.
// Box (padded cell coordinates, origin o and extents e) that the body, grown by `margin` cells, can reach at any time: the union over
// the primitives that ADD material (the first one and every union; a difference only removes) of centre +- (motion amplitude +
// extent / smallest scale of the map + margin).  A plane, or a map that can scale to nothing, reaches everywhere: the whole grid.
void wl_body_box(const wl_sim* s, float margin, int interior, int o[3], int e[3])
{
    const Grid& g = s->lev[0].g;
    const wl_config& c = s->cfg;
    for (int d = 0; d < 3; ++d) { o[d] = interior && d < s->nd ? 1 : 0; e[d] = interior ? g.n[d] : g.S[d]; }
    if (c.body.kind == WL_BODY_NONE) return;
    for (int d = 0; d < s->nd; ++d) {
        const int first = interior ? 1 : 0, last = interior ? g.n[d] : g.n[d] + 1;
        int lo = last + 1, hi = first - 1;
        bool whole = false;
        for (int k = 0; k <= c.nextra && !whole; ++k) {
            const wl_body& b = k == 0 ? c.body : c.extra[k - 1];
            if (k > 0 && c.extra_op[k - 1] != WL_OP_UNION) continue;
            if (b.kind == WL_BODY_PLANE || (b.kind == WL_BODY_CYLINDER && d == b.axis)) { whole = true; break; }   // it spans the direction
            float ext = b.R;                                      // sphere / circle / cylinder cross-section
            if (b.kind == WL_BODY_TORUS) ext = d == b.axis ? b.r : b.R + b.r;
            if (b.shell > 0.0f) ext += b.shell;
            float m = margin;
            const float smin = 1.0f - fabsf(b.scale_amp[d]);      // xi = s (x - c), s = 1 + scale_amp cos(.): x-extent = extent / s
            if (b.scale_amp[0] != 0.0f || b.scale_amp[1] != 0.0f || b.scale_amp[2] != 0.0f) {
                if (smin < 0.25f) { whole = true; break; }
                ext /= smin;
                m = 1.5f * margin + 1.0f;                         // the distance of a non-rigid map is first-order (R-E3): a generous band
            }
            float reach = ext + m;
            if (b.motion == WL_MOTION_SIN) reach += fabsf(b.amp[d]);
            const int l = (int)floorf(b.centre[d] - reach), h = (int)ceilf(b.centre[d] + reach) + 1;      // padded coordinates c = x + 1/2
            if (l < lo) lo = l;
            if (h > hi) hi = h;
        }
        if (whole) { lo = first; hi = last; }
        if (lo < first) lo = first;
        if (hi > last) hi = last;
        if (g.per[d] && (lo <= 2 || hi >= g.n[d] - 1)) { lo = first; hi = last; }   // ghosts mirror the far side: whole direction
        if (hi < lo) { lo = first; hi = last; }
        o[d] = lo; e[d] = hi - lo + 1;
    }
}

// measure! over the whole padded grid the first time; afterwards only over the box the body can reach: mu0 = 1 and
// mu1 = 0 further than eps from the surface never change (the boundary-face zeros of mu0 neither), and the supported
// motion is a sinusoidal translation of known amplitude, so the box is known on the host although t is device-resident.
void wl_k_measure(wl_sim* s)
{
    const Grid& g = s->lev[0].g;
    Tiling T = wl_tiles_padded(s, g);
    const wl_body& b = s->cfg.body;
    if (s->measured && b.kind != WL_BODY_NONE) {
        int o[3], e[3];
        wl_body_box(s, s->cfg.eps + 2.0f, 0, o, e);                   // the face positions are half a cell off the centres
        T = wl_tiling(s->nd, o, e);
    }
    for (int d = 0; d < 3; ++d) { s->mbox_lo[d] = T.o[d]; s->mbox_hi[d] = T.o[d] + T.e[d] - 1; }
    s->measured = 1;
    cudaMemsetAsync(s->ds->band_count, 0, 4 * sizeof(int), s->st);
    {
        ProfScope ps(s, WLK_MEASURE);
        if (s->nd == 3) k_measure<3><<<wl_grid(s, T), wl_block(3), 0, s->st>>>(g, T, s->body, s->ds, s->mu0, s->mu1, s->Vf, s->ds, s->band_list, s->band_cap);
        else            k_measure<2><<<wl_grid(s, T), wl_block(2), 0, s->st>>>(g, T, s->body, s->ds, s->mu0, s->mu1, s->Vf, s->ds, s->band_list, s->band_cap);
        if (s->Vf && (!g.per[0] || !g.per[1] || (s->nd == 3 && !g.per[2]))) {
            if (s->nd == 3) k_measure_wallV<3><<<s->sm_count * 2, 256, 0, s->st>>>(g, s->body, s->ds, s->Vf);
            else            k_measure_wallV<2><<<s->sm_count * 2, 256, 0, s->st>>>(g, s->body, s->ds, s->Vf);
        }
    }
    wl_k_poisson_update(s);
}

void wl_k_bc(wl_sim* s, float* u)
{
    FlowP P = wl_flowp(s);
    const Grid& g = P.g;
    int64_t total = 3 * ((int64_t)g.S[1] * g.S[2] + (int64_t)g.S[0] * g.S[2] + (s->nd == 3 ? (int64_t)g.S[0] * g.S[1] : 0));
    int blocks = (int)((total + 255) / 256);
    if (blocks > s->sm_count * 8) blocks = s->sm_count * 8;
    ProfScope ps(s, WLK_BC);
    if (s->nd == 3) k_bc<3><<<blocks, 256, 0, s->st>>>(P, u);
    else            k_bc<2><<<blocks, 256, 0, s->st>>>(P, u);
}

void wl_k_exit_bc(wl_sim* s, float* u, const float* u0)
{
    FlowP P = wl_flowp(s);
    const Grid& g = P.g;
    int cnt = g.n[1] * (s->nd == 3 ? g.n[2] : 1);
    int blocks = (cnt + 255) / 256;
    if (blocks > s->sm_count) blocks = s->sm_count;
    {
        ProfScope ps(s, WLK_EXIT_BC);
        if (s->nd == 3) k_exit_a<3><<<blocks, 256, 0, s->st>>>(P, u, u0, s->ds, s->rb);
        else            k_exit_a<2><<<blocks, 256, 0, s->st>>>(P, u, u0, s->ds, s->rb);
    }
    {
        ProfScope ps(s, WLK_EXIT_BC);
        if (s->nd == 3) k_exit_b<3><<<blocks, 256, 0, s->st>>>(P, u, s->ds);
        else            k_exit_b<2><<<blocks, 256, 0, s->st>>>(P, u, s->ds);
    }
}

void wl_k_cfl(wl_sim* s, const float* u)
{
    const Grid& g = s->lev[0].g;
    const VT& vt = s->lev[0].vt;
    const wl_config& c = s->cfg;
    ProfScope ps(s, WLK_CFL);
    if (s->nd == 3) k_cfl<3><<<wl_vgrid(s, vt), WL_VB, 0, s->st>>>(g, vt, u, s->ds, s->rb, c.nu, c.cfl_c, c.cfl_cnu, c.dt_max);
    else            k_cfl<2><<<wl_vgrid(s, vt), WL_VB, 0, s->st>>>(g, vt, u, s->ds, s->rb, c.nu, c.cfl_c, c.cfl_cnu, c.dt_max);
}

void wl_k_energy(wl_sim* s, const float* u)
{
    const Grid& g = s->lev[0].g;
    const VT& vt = s->lev[0].vt;
    ProfScope ps(s, WLK_ENERGY);
    if (s->nd == 3) k_energy<3><<<wl_vgrid(s, vt), WL_VB, 0, s->st>>>(g, vt, u, s->ds, s->rb);
    else            k_energy<2><<<wl_vgrid(s, vt), WL_VB, 0, s->st>>>(g, vt, u, s->ds, s->rb);
}

void wl_k_force(wl_sim* s, double t)
{
    const Grid& g = s->lev[0].g;
    Tiling T = wl_tiles_interior(s, g);
    if (s->cfg.body.kind != WL_BODY_NONE) {      // K(d) vanishes further than one cell from the surface: the body's box is enough
        int o[3], e[3];
        wl_body_box(s, 3.0f, 1, o, e);
        T = wl_tiling(s->nd, o, e);
    }
    {
        ProfScope ps(s, WLK_SET_TIME);
        k_force_time<<<1, 1, 0, s->st>>>(s->ds, body_all(s), t);
    }
    ProfScope ps(s, WLK_FORCE);
    if (s->nd == 3) k_force<3><<<wl_grid(s, T), wl_block(3), 0, s->st>>>(g, T, s->body, s->p, s->ds, s->rb);
    else            k_force<2><<<wl_grid(s, T), wl_block(2), 0, s->st>>>(g, T, s->body, s->p, s->ds, s->rb);
}

void wl_k_init_tgv(wl_sim* s, int sign)
{
    const Grid& g = s->lev[0].g;
    Tiling T = wl_tiles_padded(s, g);
    ProfScope ps(s, WLK_MISC);
    if (s->nd == 3) k_init_tgv<3><<<wl_grid(s, T), wl_block(3), 0, s->st>>>(g, T, s->u, s->p, sign);
    else            k_init_tgv<2><<<wl_grid(s, T), wl_block(2), 0, s->st>>>(g, T, s->u, s->p, sign);
}

void wl_k_fill(wl_sim* s, float* a, int64_t n, float v)
{
    int blocks = (int)((n + 1023) / 1024);
    if (blocks > s->sm_count * 8) blocks = s->sm_count * 8;
    if (blocks < 1) blocks = 1;
    ProfScope ps(s, WLK_MISC);
    k_fill<<<blocks, 256, 0, s->st>>>(a, n, v);
}

void wl_k_fill_u(wl_sim* s, float* u)
{
    const Grid& g = s->lev[0].g;
    for (int i = 0; i < s->nd; ++i) wl_k_fill(s, u + i * g.nalloc, g.nalloc, s->cfg.U[i]);
}

void wl_k_pack(wl_sim* s, const Grid& g, const float* padded, float* interior, int ncomp, float scale, int whole)
{
    Tiling T = whole ? wl_tiles_padded(s, g) : wl_tiles_interior(s, g);
    ProfScope ps(s, WLK_MISC);
    if (s->nd == 3) k_pack<3><<<wl_grid(s, T), wl_block(3), 0, s->st>>>(g, T, padded, interior, ncomp, scale);
    else            k_pack<2><<<wl_grid(s, T), wl_block(2), 0, s->st>>>(g, T, padded, interior, ncomp, scale);
}

void wl_k_unpack(wl_sim* s, const Grid& g, const float* interior, float* padded, int ncomp)
{
    Tiling T = wl_tiles_interior(s, g);
    ProfScope ps(s, WLK_MISC);
    if (s->nd == 3) k_unpack<3><<<wl_grid(s, T), wl_block(3), 0, s->st>>>(g, T, interior, padded, ncomp);
    else            k_unpack<2><<<wl_grid(s, T), wl_block(2), 0, s->st>>>(g, T, interior, padded, ncomp);
}
