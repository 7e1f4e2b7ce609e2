// wl_generic.cu -- the GENERIC engine of libwl: the same time step (mom_step, routine list P:139; readings of
// DESIGN.md section 3) written once over a scalar type T, one thread per cell, no tiling, no fusion.  Two instantiations:
//   T = double  the fp64 mode of the solver ("T" keyword, "T=Float32": the precision is a parameter of the paper's
//               simulation type);
//   T = Dual    value + one derivative lane d/d(theta) through EVERY kernel of the step -- measure!, conv_diff!, BDIM!, BC!,
//               exitBC!, project! (multigrid + PCG, dot products included), the force and the energy sums -- i.e. the forward-mode
//               tangent of the whole solver with respect to one parameter theta.
// The tuned fp32 kernels (wl_convdiff.cu, wl_poisson.cu, ...) are the product's hot path; this engine trades speed for generality:
// every stage is a plain kernel over the padded arrays (layout: one ghost cell per side, x fastest, idx = c0 + S0 (c1 + S1 c2)),
// reductions are two-stage with a fixed tree (bit-reproducible), the PCG scalars stay on the device.
#include <cstdio>
#include <cstring>
#include <cmath>
#include <new>
#include "wl_internal.h"
#include "wl_dual.cuh"

#define G_NT 256                 // threads per block
#define G_NB 256                 // blocks of a reducing kernel (partials per value and lane)
#define G_PI 3.14159265358979323846

struct GLev {
    int n[3], S[3], per[3];      // interior cells, padded sizes (S[2] = 1 in 2-D), periodic flags
    long long st[3], nc;         // strides, padded cell count
    int nd;
};
__host__ __device__ inline long long gl_idx(const GLev& g, int c0, int c1, int c2) { return c0 + (long long)g.S[0] * (c1 + (long long)g.S[1] * c2); }
__host__ __device__ inline void gl_coords(const GLev& g, long long k, int (&c)[3])
{
    c[0] = (int)(k % g.S[0]);
    const long long t = k / g.S[0];
    c[1] = (int)(t % g.S[1]);
    c[2] = (int)(t / g.S[1]);
}
__host__ __device__ inline bool gl_interior(const GLev& g, const int (&c)[3])
{
    for (int d = 0; d < g.nd; ++d) if (c[d] < 1 || c[d] > g.n[d]) return false;
    return true;
}
__host__ __device__ inline int gl_wrap(int c, int N, int per) { if (per) { if (c < 1) c += N; else if (c > N) c -= N; } return c; }

template <class T>
struct GPart {
    int kind, axis, motion, op, scaled;
    T centre[3], R, r, amp[3], freq[3], phase[3], shell, samp[3], sfreq, sphase, spin;
};
template <class T>
struct GBody { int n; GPart<T> part[4]; T eps; };

// device scalars (T each)
enum { GS_RHO, GS_RHO0, GS_ALPHA, GS_BETA, GS_MEAN, GS_EXIT, GS_CFL, GS_F0, GS_F1, GS_F2, GS_KE, GS_ENS, GS_RES, GS_COUNT };
enum { GF_LIVE, GF_NAN, GF_COUNT };

template <class T>
struct GEngine {
    int nd, nlev;
    GLev lev[WL_MAXLEV];
    T *u, *u0, *f, *r, *V, *mu0, *mu1, *p, *sig;
    T *L[WL_MAXLEV], *iD[WL_MAXLEV], *x[WL_MAXLEV], *rr[WL_MAXLEV], *e[WL_MAXLEV], *q[WL_MAXLEV];
    T* sc;                       // [GS_COUNT]
    int* flags;                  // [GF_COUNT]
    double* partial;             // [4 values][2 lanes][G_NB]
    T* hsc;                      // pinned host mirror of sc
    int* hflags;
    GBody<T> body;
    T nu, U[3], eps;
    int exit_bc;
    cudaStream_t st;
};

// ------------------------------------------------------------------ reductions: block tree -> partial; one block finishes
template <class T, int NV>
__device__ inline void g_block_partial(const T (&v)[NV], double* partial)
{
    __shared__ double sm[G_NT];
    const int tid = threadIdx.x;
    for (int k = 0; k < NV; ++k)
        for (int l = 0; l < Lanes<T>::N; ++l) {
            sm[tid] = Lanes<T>::get(v[k], l);
            __syncthreads();
            for (int o = G_NT / 2; o > 0; o >>= 1) {
                if (tid < o) sm[tid] += sm[tid + o];
                __syncthreads();
            }
            if (tid == 0) partial[(k * 2 + l) * G_NB + blockIdx.x] = sm[0];
            __syncthreads();
        }
}
// max instead of sum (CFL): lane 0 only
__device__ inline void g_block_partial_max(double v, double* partial)
{
    __shared__ double sm[G_NT];
    const int tid = threadIdx.x;
    sm[tid] = v;
    __syncthreads();
    for (int o = G_NT / 2; o > 0; o >>= 1) {
        if (tid < o) sm[tid] = sm[tid] > sm[tid + o] ? sm[tid] : sm[tid + o];
        __syncthreads();
    }
    if (tid == 0) partial[blockIdx.x] = sm[0];
}
// called by every thread of ONE block of G_NT threads: the totals of NV values (fixed tree over the G_NB partials)
template <class T, int NV>
__device__ inline void g_finish(const double* partial, T (&out)[NV])
{
    __shared__ double sm[G_NT];
    const int tid = threadIdx.x;
    for (int k = 0; k < NV; ++k) {
        double l2[2] = { 0.0, 0.0 };
        for (int l = 0; l < Lanes<T>::N; ++l) {
            sm[tid] = tid < G_NB ? partial[(k * 2 + l) * G_NB + tid] : 0.0;
            __syncthreads();
            for (int o = G_NT / 2; o > 0; o >>= 1) {
                if (tid < o) sm[tid] += sm[tid + o];
                __syncthreads();
            }
            l2[l] = sm[0];
            __syncthreads();
        }
        out[k] = Lanes<T>::make(l2);
    }
}

// ------------------------------------------------------------------ body: kernel moments, SDF, map (R-B, R-E, R-E3)
template <class T> __device__ inline T g_K(T s, T eps) { if (g_abs(s) >= eps) return T(0.0); return (T(1.0) + g_cos(T(G_PI) * s / eps)) / (T(2.0) * eps); }
template <class T> __device__ inline T g_mu0(T d, T eps)
{
    const T a = d / eps;
    if (a <= T(-1.0)) return T(0.0);
    if (a >= T(1.0)) return T(1.0);
    return T(0.5) + T(0.5) * a + g_sin(T(G_PI) * a) / T(2.0 * G_PI);
}
template <class T> __device__ inline T g_mu1(T d, T eps)
{
    const T a = d / eps;
    if (a <= T(-1.0) || a >= T(1.0)) return T(0.0);
    return eps * (T(0.25) - T(0.25) * a * a - (a * g_sin(T(G_PI) * a) + (T(1.0) + g_cos(T(G_PI) * a)) / T(G_PI)) / T(2.0 * G_PI));
}

template <class T>
__device__ inline T g_prim(int nd, const GPart<T>& p, const T (&xi)[3], T (&g)[3])
{
    g[0] = g[1] = g[2] = T(0.0);
    if (p.kind == WL_BODY_SPHERE) {
        T rr = T(0.0);
        for (int k = 0; k < nd; ++k) rr += xi[k] * xi[k];
        rr = g_sqrt(rr);
        if (g_val(rr) >= 1e-12) for (int k = 0; k < nd; ++k) g[k] = xi[k] / rr;
        return rr - p.R;
    }
    if (p.kind == WL_BODY_PLANE) { g[p.axis] = T(1.0); return xi[p.axis]; }
    const int a = p.axis, b = (a + 1) % 3, c = (a + 2) % 3;
    const T rho = g_sqrt(xi[b] * xi[b] + xi[c] * xi[c]);
    if (p.kind == WL_BODY_CYLINDER) {
        if (g_val(rho) >= 1e-12) { g[b] = xi[b] / rho; g[c] = xi[c] / rho; }
        return rho - p.R;
    }
    const T w = rho - p.R;
    const T q = g_sqrt(w * w + xi[a] * xi[a]);
    if (g_val(q) >= 1e-12 && g_val(rho) >= 1e-12) {
        g[a] = xi[a] / q; g[b] = (w / q) * (xi[b] / rho); g[c] = (w / q) * (xi[c] / rho);
    } else if (g_val(q) >= 1e-12) {
        g[a] = xi[a] / q;
    }
    return q - p.r;
}

template <class T>
__device__ inline T g_body_eval(int nd, const GBody<T>& B, const double (&x)[3], T t, T (&nrm)[3], T (&vel)[3])
{
    T d = T(1e30);
    nrm[0] = nrm[1] = nrm[2] = T(0.0);
    vel[0] = vel[1] = vel[2] = T(0.0);
    for (int e = 0; e < B.n; ++e) {
        const GPart<T>& p = B.part[e];
        T c[3], cdot[3], s[3], sdot[3], rel[3], xi[3], g[3];
        const T phs = T(2.0 * G_PI) * p.sfreq * t + p.sphase;
        for (int k = 0; k < 3; ++k) {
            c[k] = p.centre[k]; cdot[k] = T(0.0);
            if (p.motion == WL_MOTION_SIN && k < nd) {
                const T ph = T(2.0 * G_PI) * p.freq[k] * t + p.phase[k];
                c[k] = c[k] + p.amp[k] * g_sin(ph);
                cdot[k] = p.amp[k] * T(2.0 * G_PI) * p.freq[k] * g_cos(ph);
            }
            s[k] = k < nd ? T(1.0) + p.samp[k] * g_cos(phs) : T(1.0);
            sdot[k] = k < nd ? -(p.samp[k] * T(2.0 * G_PI) * p.sfreq * g_sin(phs)) : T(0.0);
            rel[k] = k < nd ? T(x[k]) - c[k] : T(0.0);
            xi[k] = s[k] * rel[k];
        }
        T d0 = g_prim<T>(nd, p, xi, g);
        if (g_val(p.shell) > 0.0) {
            const bool neg = g_val(d0) < 0.0;
            d0 = g_abs(d0) - p.shell;
            if (neg) for (int k = 0; k < 3; ++k) g[k] = -g[k];
        }
        if (p.scaled) {
            T m = T(0.0);
            for (int k = 0; k < nd; ++k) { g[k] = g[k] * s[k]; m += g[k] * g[k]; }
            m = g_sqrt(m);
            if (g_val(m) >= 1e-12) {
                d0 = d0 / m;
                for (int k = 0; k < nd; ++k) g[k] = g[k] / m;
            } else {
                g[0] = g[1] = g[2] = T(0.0);
            }
        }
        if (p.op == 1) { d0 = -d0; for (int k = 0; k < 3; ++k) g[k] = -g[k]; }
        const bool take = e == 0 || (p.op == 1 ? g_val(d0) > g_val(d) : g_val(d0) < g_val(d));
        if (take) {
            d = d0;
            for (int k = 0; k < 3; ++k) { nrm[k] = g[k]; vel[k] = T(0.0); }
            for (int k = 0; k < nd; ++k) vel[k] = cdot[k] - (sdot[k] / s[k]) * rel[k];
            if (g_val(p.spin) != 0.0 || g_der(p.spin) != 0.0) {
                const int a = nd == 3 ? p.axis : 2, b1 = (a + 1) % 3, c1 = (a + 2) % 3;
                if (b1 < nd) vel[b1] = vel[b1] - p.spin * rel[c1];
                if (c1 < nd) vel[c1] = vel[c1] + p.spin * rel[b1];
            }
        }
    }
    return d;
}

// ------------------------------------------------------------------ measure! (O2)
template <class T>
__global__ void g_measure(GLev g, GBody<T> B, T t, T* mu0, T* mu1, T* V)
{
    const int nd = g.nd;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        for (int i = 0; i < nd; ++i) {
            double xf[3] = { 0.0, 0.0, 0.0 };
            for (int d = 0; d < nd; ++d) xf[d] = c[d] - 0.5;
            xf[i] -= 0.5;
            T m0 = T(1.0), m1 = T(0.0), nrm[3] = { T(0.0), T(0.0), T(0.0) }, vel[3] = { T(0.0), T(0.0), T(0.0) };
            if (B.n > 0) {
                const T d = g_body_eval<T>(nd, B, xf, t, nrm, vel);
                m0 = g_mu0<T>(d, B.eps);
                m1 = g_mu1<T>(d, B.eps);
            }
            mu0[i * g.nc + k] = m0;
            for (int j = 0; j < nd; ++j) mu1[(i * nd + j) * g.nc + k] = m1 * nrm[j];
            V[i * g.nc + k] = vel[i];
        }
    }
}

// ghost planes of `ncomp` arrays in direction j: periodic wrap (mode 0); mu0 = 0 on the two boundary-normal faces of
// component j in a non-periodic direction (mode 1, R-O)
template <class T>
__global__ void g_planes(GLev g, T* a, int ncomp, int j, int mode)
{
    const int d0 = j == 0 ? 1 : 0, d1 = j == 2 ? 1 : 2;
    const long long A = (long long)g.S[d0] * g.S[d1];
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < A * ncomp; k += (long long)gridDim.x * blockDim.x) {
        const int m = (int)(k / A);
        const long long ab = k % A;
        int c[3] = { 0, 0, 0 };
        c[d0] = (int)(ab % g.S[d0]); c[d1] = (int)(ab / g.S[d0]);
        if (g.nd == 2) c[2] = 0;
        const long long b = gl_idx(g, c[0], c[1], c[2]);     // c_j = 0
        T* arr = a + m * g.nc;
        const int N = g.n[j];
        if (mode == 0) {
            arr[b] = arr[b + N * g.st[j]];
            arr[b + (N + 1) * g.st[j]] = arr[b + g.st[j]];
        } else if (m == 0) {
            arr[b + g.st[j]] = T(0.0);
            arr[b + (N + 1) * g.st[j]] = T(0.0);
        }
    }
}

// BC! (O5) for direction j over the whole padded range of the others
template <class T>
__global__ void g_bc(GLev g, T* u, int j, T Uj, int exit_bc)
{
    const int nd = g.nd;
    const int d0 = j == 0 ? 1 : 0, d1 = j == 2 ? 1 : 2;
    const long long A = (long long)g.S[d0] * g.S[d1];
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < A * nd; k += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(k / A);
        const long long ab = k % A;
        int c[3] = { 0, 0, 0 };
        c[d0] = (int)(ab % g.S[d0]); c[d1] = (int)(ab / g.S[d0]);
        if (nd == 2) c[2] = 0;
        const long long b = gl_idx(g, c[0], c[1], c[2]);
        T* a = u + i * g.nc;
        const int N = g.n[j];
        const long long sj = g.st[j];
        if (g.per[j]) { a[b] = a[b + N * sj]; a[b + (N + 1) * sj] = a[b + sj]; }
        else if (i == j) { a[b] = Uj; a[b + sj] = Uj; if (!(exit_bc && j == 0)) a[b + (N + 1) * sj] = Uj; }
        else { a[b] = a[b + sj]; a[b + (N + 1) * sj] = a[b + N * sj]; }
    }
}

// exitBC! (O6): pass 0 advects and accumulates the plane sum, pass 1 (one block) forms the correction, pass 2 applies it
template <class T>
__global__ void g_exit_a(GLev g, T* u, const T* u0, T U0, T dt, double* partial)
{
    const int n1 = g.n[1], n2 = g.nd == 3 ? g.n[2] : 1;
    T v[1] = { T(0.0) };
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n1 * n2; t += gridDim.x * blockDim.x) {
        const int c1 = 1 + t % n1, c2 = g.nd == 3 ? 1 + t / n1 : 0;
        const long long id = gl_idx(g, g.n[0] + 1, c1, c2);
        const T val = u0[id] - U0 * dt * (u0[id] - u0[id - 1]);
        u[id] = val;
        v[0] += val;
    }
    g_block_partial<T, 1>(v, partial);
}
template <class T>
__global__ void g_exit_b(GLev g, const double* partial, T U0, T* sc)
{
    T v[1];
    g_finish<T, 1>(partial, v);
    if (threadIdx.x == 0) sc[GS_EXIT] = v[0] / T((double)(g.n[1] * (g.nd == 3 ? g.n[2] : 1))) - U0;
}
template <class T>
__global__ void g_exit_c(GLev g, T* u, const T* sc)
{
    const int n1 = g.n[1], n2 = g.nd == 3 ? g.n[2] : 1;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n1 * n2; t += gridDim.x * blockDim.x) {
        const int c1 = 1 + t % n1, c2 = g.nd == 3 ? 1 + t / n1 : 0;
        u[gl_idx(g, g.n[0] + 1, c1, c2)] -= sc[GS_EXIT];
    }
}

// ------------------------------------------------------------------ conv_diff! (O3)
template <class T> __device__ inline T g_med3(T a, T b, T c)
{
    const T lo = a < b ? a : b, hi = a < b ? b : a;
    return c < lo ? lo : (c > hi ? hi : c);
}
template <class T> __device__ inline T g_quick(T U, T C, T D)
{
    return g_med3<T>((T(5.0) * C + T(2.0) * D - U) / T(6.0), C, g_med3<T>(T(10.0) * C - T(9.0) * U, C, D));
}
template <class T>
__device__ inline T g_W(const GLev& g, const T* w, int comp, int c0, int c1, int c2)
{
    c0 = gl_wrap(c0, g.n[0], g.per[0]);
    c1 = gl_wrap(c1, g.n[1], g.per[1]);
    if (g.nd == 3) c2 = gl_wrap(c2, g.n[2], g.per[2]);
    return w[comp * g.nc + gl_idx(g, c0, c1, c2)];
}
// flux through the LOWER j-boundary of the control volume of w_i at c
template <class T>
__device__ inline T g_flux(const GLev& g, const T* w, T nu, int i, int j, const int (&c)[3])
{
    int di[3] = { 0, 0, 0 }, dj[3] = { 0, 0, 0 };
    di[i] = 1; dj[j] = 1;
    const int N = g.n[j], per = g.per[j];
    const T phi = T(0.5) * (g_W<T>(g, w, j, c[0] - di[0], c[1] - di[1], c[2] - di[2]) + g_W<T>(g, w, j, c[0], c[1], c[2]));
    const T wc = g_W<T>(g, w, i, c[0], c[1], c[2]);
    const T wm = g_W<T>(g, w, i, c[0] - dj[0], c[1] - dj[1], c[2] - dj[2]);
    T psi;
    if (g_val(phi) > 0.0) {
        if (!per && c[j] <= 1 + (i == j ? 1 : 0)) psi = T(0.5) * (wm + wc);
        else psi = g_quick<T>(g_W<T>(g, w, i, c[0] - 2 * dj[0], c[1] - 2 * dj[1], c[2] - 2 * dj[2]), wm, wc);
    } else {
        if (!per && c[j] == N + 1) psi = T(0.5) * (wm + wc);
        else psi = g_quick<T>(g_W<T>(g, w, i, c[0] + dj[0], c[1] + dj[1], c[2] + dj[2]), wc, wm);
    }
    return phi * psi - nu * (wc - wm);
}
// f = u0 + dt r - V on the whole padded array, r = conv_diff(w) on the interior and 0 in the ghosts (O3 + first half of O4)
template <class T>
__global__ void g_convdiff_f(GLev g, const T* w, const T* u0, const T* V, T nu, T dt, T* f)
{
    const int nd = g.nd;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        const bool in = gl_interior(g, c);
        for (int i = 0; i < nd; ++i) {
            T acc = T(0.0);
            if (in)
                for (int j = 0; j < nd; ++j) {
                    int cp[3] = { c[0], c[1], c[2] };
                    cp[j] += 1;
                    acc += g_flux<T>(g, w, nu, i, j, c) - g_flux<T>(g, w, nu, i, j, cp);
                }
            f[i * g.nc + k] = u0[i * g.nc + k] + dt * acc - V[i * g.nc + k];
        }
    }
}
// BDIM! + scale_u! (second half of O4): B = V + mu0 f + sum_j mu1_ij (f[c+dj] - f[c-dj])/2
template <class T>
__global__ void g_bdim(GLev g, const T* f, const T* V, const T* mu0, const T* mu1, T* u, int corr)
{
    const int nd = g.nd;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        for (int i = 0; i < nd; ++i) {
            T B = V[i * g.nc + k] + mu0[i * g.nc + k] * f[i * g.nc + k];
            for (int j = 0; j < nd; ++j)
                B += mu1[(i * nd + j) * g.nc + k] * T(0.5) * (f[i * g.nc + k + g.st[j]] - f[i * g.nc + k - g.st[j]]);
            u[i * g.nc + k] = corr ? T(0.5) * (u[i * g.nc + k] + B) : B;
        }
    }
}

// ------------------------------------------------------------------ Poisson operator, multigrid (O7, O8)
template <class T>
__global__ void g_diag(GLev g, const T* L, T* iD)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) { iD[k] = T(0.0); continue; }
        T D = T(0.0);
        for (int i = 0; i < g.nd; ++i) D -= L[i * g.nc + k] + L[i * g.nc + k + g.st[i]];
        iD[k] = fabs(g_val(D)) > 2.0 * g.nd * 1e-6 ? T(1.0) / D : T(0.0);
    }
}
template <class T>
__global__ void g_restrict_L(GLev gf, GLev gc, const T* Lf, T* Lc)
{
    const int nd = gc.nd;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < gc.nc; k += (long long)gridDim.x * blockDim.x) {
        int C[3];
        gl_coords(gc, k, C);
        for (int i = 0; i < nd; ++i) {
            bool ok = C[i] >= 1 && C[i] <= gc.n[i] + 1;
            for (int d = 0; d < nd; ++d) if (d != i && (C[d] < 1 || C[d] > gc.n[d])) ok = false;
            if (!ok) { Lc[i * gc.nc + k] = T(0.0); continue; }
            const int b[3] = { 2 * C[0] - 1, 2 * C[1] - 1, nd == 3 ? 2 * C[2] - 1 : 0 };
            T sum = T(0.0);
            for (int a2 = 0; a2 < (nd == 3 ? 2 : 1); ++a2)
                for (int a1 = 0; a1 < 2; ++a1)
                    for (int a0 = 0; a0 < 2; ++a0) {
                        const int a[3] = { a0, a1, a2 };
                        if (a[i] != 0) continue;
                        sum += Lf[i * gf.nc + gl_idx(gf, b[0] + a0, b[1] + a1, b[2] + a2)];
                    }
            Lc[i * gc.nc + k] = T(0.5) * sum;
        }
    }
}
// q = A e on the interior (periodic neighbours by index wrap), partial sum of q.e
template <class T>
__device__ inline T g_Ae(const GLev& g, const T* L, const T* e, long long k, const int (&c)[3])
{
    T acc = T(0.0);
    for (int i = 0; i < g.nd; ++i) {
        int cl[3] = { c[0], c[1], c[2] }, ch[3] = { c[0], c[1], c[2] };
        cl[i] = gl_wrap(c[i] - 1, g.n[i], g.per[i]);
        ch[i] = gl_wrap(c[i] + 1, g.n[i], g.per[i]);
        const T el = e[gl_idx(g, cl[0], cl[1], cl[2])], eh = e[gl_idx(g, ch[0], ch[1], ch[2])];
        acc += L[i * g.nc + k + g.st[i]] * (eh - e[k]) - L[i * g.nc + k] * (e[k] - el);
    }
    return acc;
}
template <class T>
__global__ void g_matvec(GLev g, const T* L, const T* e, T* q, const int* flags, double* partial)
{
    T v[1] = { T(0.0) };
    if (flags[GF_LIVE])
        for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
            int c[3];
            gl_coords(g, k, c);
            if (!gl_interior(g, c)) continue;
            const T a = g_Ae<T>(g, L, e, k, c);
            q[k] = a;
            v[0] += a * e[k];
        }
    g_block_partial<T, 1>(v, partial);
}
// level-0 residual r = sig - A x (no guard)
template <class T>
__global__ void g_residual(GLev g, const T* L, const T* x, const T* sig, T* r)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        r[k] = sig[k] - g_Ae<T>(g, L, x, k, c);
    }
}
// PCG, stage by stage (R-T, R-T2)
template <class T>
__global__ void g_pcg_mean_a(GLev g, const T* r, const T* iD, double* partial)
{
    T v[2] = { T(0.0), T(0.0) };
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c) || g_val(iD[k]) == 0.0) continue;
        v[0] += r[k]; v[1] += T(1.0);
    }
    g_block_partial<T, 2>(v, partial);
}
template <class T>
__global__ void g_pcg_mean_b(const double* partial, T* sc)
{
    T v[2];
    g_finish<T, 2>(partial, v);
    if (threadIdx.x == 0) sc[GS_MEAN] = g_val(v[1]) > 0.0 ? v[0] / v[1] : T(0.0);
}
// r -= mean on the coupled cells; z = e = iD r; partial rho = r.z
template <class T>
__global__ void g_pcg_init(GLev g, T* r, const T* iD, T* e, const T* sc, double* partial)
{
    T v[1] = { T(0.0) };
    const T m = sc[GS_MEAN];
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        if (g_val(iD[k]) != 0.0) r[k] -= m;
        const T z = iD[k] * r[k];
        e[k] = z;
        v[0] += z * r[k];
    }
    g_block_partial<T, 1>(v, partial);
}
template <class T>
__global__ void g_pcg_rho0(const double* partial, T* sc, int* flags)
{
    T v[1];
    g_finish<T, 1>(partial, v);
    if (threadIdx.x == 0) { sc[GS_RHO] = v[0]; sc[GS_RHO0] = v[0]; flags[GF_LIVE] = fabs(g_val(v[0])) < WL_TAU ? 0 : 1; }
}
template <class T>
__global__ void g_pcg_alpha(const double* partial, T* sc, int* flags)
{
    T v[1];
    g_finish<T, 1>(partial, v);
    if (threadIdx.x == 0 && flags[GF_LIVE]) {
        const double gm = g_val(v[0]);
        if (gm == 0.0 || !isfinite(gm)) flags[GF_LIVE] = 0;
        else sc[GS_ALPHA] = sc[GS_RHO] / v[0];
    }
}
// x += alpha e; r -= alpha q; partial rho' = r.(iD r)
template <class T>
__global__ void g_pcg_update(GLev g, T* x, T* r, const T* e, const T* q, const T* iD, const T* sc, const int* flags, double* partial)
{
    T v[1] = { T(0.0) };
    if (flags[GF_LIVE]) {
        const T alpha = sc[GS_ALPHA];
        for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
            int c[3];
            gl_coords(g, k, c);
            if (!gl_interior(g, c)) continue;
            x[k] += alpha * e[k];
            r[k] -= alpha * q[k];
            v[0] += (iD[k] * r[k]) * r[k];
        }
    }
    g_block_partial<T, 1>(v, partial);
}
template <class T>
__global__ void g_pcg_beta(const double* partial, T* sc, int* flags)
{
    T v[1];
    g_finish<T, 1>(partial, v);
    if (threadIdx.x == 0 && flags[GF_LIVE]) {
        const double r2 = g_val(v[0]);
        if (fabs(r2) < WL_TAU || fabs(r2) < WL_THETA * fabs(g_val(sc[GS_RHO0]))) flags[GF_LIVE] = 0;
        else { sc[GS_BETA] = v[0] / sc[GS_RHO]; sc[GS_RHO] = v[0]; }
    }
}
template <class T>
__global__ void g_pcg_dir(GLev g, T* e, const T* r, const T* iD, const T* sc, const int* flags)
{
    if (!flags[GF_LIVE]) return;
    const T beta = sc[GS_BETA];
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        e[k] = beta * e[k] + iD[k] * r[k];
    }
}
template <class T>
__global__ void g_restrict_r(GLev gf, GLev gc, const T* rf, T* rc, T* xc)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < gc.nc; k += (long long)gridDim.x * blockDim.x) {
        int C[3];
        gl_coords(gc, k, C);
        xc[k] = T(0.0);
        if (!gl_interior(gc, C)) { rc[k] = T(0.0); continue; }
        T s = T(0.0);
        for (int a2 = 0; a2 < (gc.nd == 3 ? 2 : 1); ++a2)
            for (int a1 = 0; a1 < 2; ++a1)
                for (int a0 = 0; a0 < 2; ++a0)
                    s += rf[gl_idx(gf, 2 * C[0] - 1 + a0, 2 * C[1] - 1 + a1, gc.nd == 3 ? 2 * C[2] - 1 + a2 : 0)];
        rc[k] = s;
    }
}
// e = P x_c into the fine e array (interior), then x_f += e and r_f -= A e
template <class T>
__global__ void g_prolong_a(GLev gf, GLev gc, const T* xc, T* ef)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < gf.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(gf, k, c);
        if (!gl_interior(gf, c)) { ef[k] = T(0.0); continue; }
        ef[k] = xc[gl_idx(gc, (c[0] + 1) / 2, (c[1] + 1) / 2, gf.nd == 3 ? (c[2] + 1) / 2 : 0)];
    }
}
template <class T>
__global__ void g_prolong_b(GLev g, const T* L, const T* e, T* x, T* r)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        x[k] += e[k];
        r[k] -= g_Ae<T>(g, L, e, k, c);
    }
}
// project!: sig = div u, x = sc p  /  u -= L grad x, p = x / sc
template <class T>
__global__ void g_div_scale(GLev g, const T* u, const T* p, T scl, T* sig, T* x)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        x[k] = scl * p[k];
        if (!gl_interior(g, c)) { sig[k] = T(0.0); continue; }
        T d = T(0.0);
        for (int i = 0; i < g.nd; ++i) d += u[i * g.nc + k + g.st[i]] - u[i * g.nc + k];
        sig[k] = d;
    }
}
template <class T>
__global__ void g_gradient(GLev g, T* u, const T* L, const T* x, T* p, T scl)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        p[k] = x[k] / scl;
        if (!gl_interior(g, c)) continue;
        for (int i = 0; i < g.nd; ++i) {
            int cl[3] = { c[0], c[1], c[2] };
            cl[i] = gl_wrap(c[i] - 1, g.n[i], g.per[i]);
            u[i * g.nc + k] -= L[i * g.nc + k] * (x[k] - x[gl_idx(g, cl[0], cl[1], cl[2])]);
        }
    }
}
template <class T>
__global__ void g_resmax_a(GLev g, const T* r, double* partial)
{
    double m = 0.0;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        const double a = fabs(g_val(r[k]));
        if (a > m || a != a) m = a;
    }
    g_block_partial_max(m, partial);
}
template <class T>
__global__ void g_max_b(const double* partial, T* sc, int slot)
{
    __shared__ double sm[G_NT];
    const int tid = threadIdx.x;
    sm[tid] = tid < G_NB ? partial[tid] : 0.0;
    __syncthreads();
    for (int o = G_NT / 2; o > 0; o >>= 1) {
        if (tid < o) sm[tid] = sm[tid] > sm[tid + o] || sm[tid] != sm[tid] ? sm[tid] : sm[tid + o];
        __syncthreads();
    }
    if (tid == 0) sc[slot] = T(sm[0]);
}

// ------------------------------------------------------------------ CFL!, force, energy (O10, O11, R-E2)
template <class T>
__global__ void g_cfl_a(GLev g, const T* u, double* partial, int* flags)
{
    double m = 0.0;
    bool bad = false;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        double a = 0.0;
        for (int i = 0; i < g.nd; ++i) {
            const double up = g_val(u[i * g.nc + k + g.st[i]]), lo = g_val(u[i * g.nc + k]);
            a += (up > 0.0 ? up : 0.0) + (lo < 0.0 ? -lo : 0.0);
            bad = bad || !isfinite(up) || !isfinite(lo);
        }
        if (a > m) m = a;
    }
    if (bad) flags[GF_NAN] = 1;
    g_block_partial_max(m, partial);
}
template <class T>
__global__ void g_force_a(GLev g, GBody<T> B, T t, const T* p, double* partial)
{
    T v[3] = { T(0.0), T(0.0), T(0.0) };
    if (B.n > 0)
        for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
            int c[3];
            gl_coords(g, k, c);
            if (!gl_interior(g, c)) continue;
            double xc[3] = { 0.0, 0.0, 0.0 };
            for (int d = 0; d < g.nd; ++d) xc[d] = c[d] - 0.5;
            T nrm[3], vel[3];
            const T d = g_body_eval<T>(g.nd, B, xc, t, nrm, vel);
            const T kk = g_K<T>(d, T(1.0));
            if (g_val(kk) == 0.0 && g_der(kk) == 0.0) continue;
            const T pk = p[k] * kk;
            for (int i = 0; i < 3; ++i) v[i] -= pk * nrm[i];
        }
    g_block_partial<T, 3>(v, partial);
}
template <class T>
__global__ void g_sum_b(const double* partial, T* sc, int slot, int nv)
{
    T v[3];
    g_finish<T, 3>(partial, v);
    if (threadIdx.x == 0) for (int k = 0; k < nv; ++k) sc[slot + k] = v[k];
}
template <class T>
__global__ void g_energy_a(GLev g, const T* u, double* partial)
{
    T v[3] = { T(0.0), T(0.0), T(0.0) };
    const int nd = g.nd;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        if (!gl_interior(g, c)) continue;
        for (int i = 0; i < nd; ++i) v[0] += T(0.5) * u[i * g.nc + k] * u[i * g.nc + k];
        for (int kk = (nd == 3 ? 0 : 2); kk < 3; ++kk) {
            const int i = (kk + 1) % 3, j = (kk + 2) % 3;
            const T w = (u[j * g.nc + k] - u[j * g.nc + k - g.st[i]]) - (u[i * g.nc + k] - u[i * g.nc + k - g.st[j]]);
            v[1] += T(0.5) * w * w;
        }
    }
    g_block_partial<T, 3>(v, partial);
}

// ------------------------------------------------------------------ initial conditions, I/O
template <class T>
__global__ void g_fill(T* a, long long n, T v) { for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) a[k] = v; }
template <class T>
__global__ void g_init_tgv(GLev g, T* u, T* p, int sign)
{
    const double k0 = (g.per[0] ? 2.0 : 1.0) * G_PI / g.n[0], k1 = (g.per[1] ? 2.0 : 1.0) * G_PI / g.n[1];
    const double k2 = g.nd == 3 ? (g.per[2] ? 2.0 : 1.0) * G_PI / g.n[2] : 0.0;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < g.nc; k += (long long)gridDim.x * blockDim.x) {
        int c[3];
        gl_coords(g, k, c);
        const double xc = c[0] - 0.5, yc = c[1] - 0.5, zc = g.nd == 3 ? c[2] - 0.5 : 0.0;
        const double cz = g.nd == 3 ? cos(k2 * zc) : 1.0;
        u[k] = T(sign * sin(k0 * (xc - 0.5)) * cos(k1 * yc) * cz);
        u[g.nc + k] = T(-sign * cos(k0 * xc) * sin(k1 * (yc - 0.5)) * cz);
        if (g.nd == 3) u[2 * g.nc + k] = T(0.0);
        p[k] = T(0.0);
    }
}
// interior of `ncomp` arrays <-> dense user buffer of `F` (float or double); lane 0 value, 1 derivative
template <class T, class F>
__global__ void g_pack(GLev g, const T* a, F* out, int ncomp, int lane)
{
    const long long ni = (long long)g.n[0] * g.n[1] * g.n[2];
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < ni * ncomp; k += (long long)gridDim.x * blockDim.x) {
        const int m = (int)(k / ni);
        long long q = k % ni;
        const int c0 = (int)(q % g.n[0]); q /= g.n[0];
        const int c1 = (int)(q % g.n[1]), c2 = (int)(q / g.n[1]);
        const T v = a[m * g.nc + gl_idx(g, c0 + 1, c1 + 1, g.nd == 3 ? c2 + 1 : 0)];
        out[k] = (F)(lane ? g_der(v) : g_val(v));
    }
}
template <class T, class F>
__global__ void g_unpack(GLev g, const F* in, T* a, int ncomp)
{
    const long long ni = (long long)g.n[0] * g.n[1] * g.n[2];
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < ni * ncomp; k += (long long)gridDim.x * blockDim.x) {
        const int m = (int)(k / ni);
        long long q = k % ni;
        const int c0 = (int)(q % g.n[0]); q /= g.n[0];
        const int c1 = (int)(q % g.n[1]), c2 = (int)(q / g.n[1]);
        a[m * g.nc + gl_idx(g, c0 + 1, c1 + 1, g.nd == 3 ? c2 + 1 : 0)] = T((double)in[k]);
    }
}

// ================================================================== host side
template <class T> T seeded(double v, bool seed);
template <> inline double seeded<double>(double v, bool) { return v; }
template <> inline Dual seeded<Dual>(double v, bool seed) { return Dual(v, seed ? 1.0 : 0.0); }

static int g_blocks(long long n) { long long b = (n + G_NT - 1) / G_NT; return (int)(b < 1 ? 1 : (b > 4096 ? 4096 : b)); }

template <class T>
static GLev make_lev(int nd, const int* n, const int* per)
{
    GLev g;
    g.nd = nd;
    for (int d = 0; d < 3; ++d) { g.n[d] = d < nd ? n[d] : 1; g.S[d] = d < nd ? n[d] + 2 : 1; g.per[d] = d < nd ? (per[d] ? 1 : 0) : 0; }
    g.st[0] = 1; g.st[1] = g.S[0]; g.st[2] = nd == 3 ? (long long)g.S[0] * g.S[1] : 0;
    g.nc = (long long)g.S[0] * g.S[1] * g.S[2];
    return g;
}

static int gen_levels(const wl_config* c, int dims[WL_MAXLEV][3])
{
    int nd = c->ndim, n[3] = { c->dims[0], c->dims[1], nd == 3 ? c->dims[2] : 1 };
    int cap = c->mg.max_levels > 0 ? c->mg.max_levels : WL_MAXLEV;
    if (cap > WL_MAXLEV) cap = WL_MAXLEV;
    int nlev = 0;
    for (;;) {
        for (int d = 0; d < 3; ++d) dims[nlev][d] = n[d];
        ++nlev;
        if (nlev >= cap) break;
        int ok = 1;
        for (int d = 0; d < nd; ++d) if ((n[d] & 1) || n[d] <= 4) ok = 0;
        if (!ok) break;
        for (int d = 0; d < nd; ++d) n[d] /= 2;
    }
    return nlev;
}

struct GCarver { char* base; size_t off; void* take(size_t b) { void* p = base ? base + off : nullptr; off += (b + 255) / 256 * 256; return p; } };

template <class T>
static size_t gen_layout(GEngine<T>* E, const wl_config* c, void* base)
{
    GCarver cv = { (char*)base, 0 };
    int nd = c->ndim, dims[WL_MAXLEV][3];
    const int nlev = gen_levels(c, dims);
    GLev g0 = make_lev<T>(nd, dims[0], c->periodic);
    const size_t sc0 = sizeof(T) * (size_t)g0.nc;
    T* sc = (T*)cv.take(sizeof(T) * GS_COUNT);
    int* flags = (int*)cv.take(sizeof(int) * GF_COUNT);
    double* partial = (double*)cv.take(sizeof(double) * 8 * G_NB);
    T* u = (T*)cv.take(sc0 * nd); T* u0 = (T*)cv.take(sc0 * nd); T* f = (T*)cv.take(sc0 * nd);
    T* V = (T*)cv.take(sc0 * nd); T* mu0 = (T*)cv.take(sc0 * nd); T* mu1 = (T*)cv.take(sc0 * nd * nd);
    T* p = (T*)cv.take(sc0); T* sig = (T*)cv.take(sc0);
    if (E) {
        E->nd = nd; E->nlev = nlev; E->sc = sc; E->flags = flags; E->partial = partial;
        E->u = u; E->u0 = u0; E->f = f; E->r = nullptr; E->V = V; E->mu0 = mu0; E->mu1 = mu1; E->p = p; E->sig = sig;
    }
    for (int l = 0; l < nlev; ++l) {
        GLev g = make_lev<T>(nd, dims[l], c->periodic);
        const size_t s1 = sizeof(T) * (size_t)g.nc;
        T* L = l == 0 ? mu0 : (T*)cv.take(s1 * nd);
        T* iD = (T*)cv.take(s1); T* x = (T*)cv.take(s1); T* r = (T*)cv.take(s1); T* e = (T*)cv.take(s1); T* q = (T*)cv.take(s1);
        if (E) { E->lev[l] = g; E->L[l] = L; E->iD[l] = iD; E->x[l] = x; E->rr[l] = r; E->e[l] = e; E->q[l] = q; }
    }
    return cv.off;
}

template <class T>
static GPart<T> make_part(const wl_body& b, int op, const wl_config* c, int which)
{
    const int sp = c->tangent_param, si = c->tangent_index;
    GPart<T> p;
    p.kind = b.kind; p.axis = b.axis; p.motion = b.motion; p.op = op;
    p.scaled = b.scale_amp[0] != 0.0f || b.scale_amp[1] != 0.0f || b.scale_amp[2] != 0.0f;
    const bool me = which == (sp == WL_SEED_SPIN ? si : 0);          // body parameters other than spin seed the FIRST primitive
    for (int k = 0; k < 3; ++k) {
        p.centre[k] = seeded<T>(b.centre[k], me && sp == WL_SEED_CENTRE && si == k);
        p.amp[k] = seeded<T>(b.amp[k], me && sp == WL_SEED_AMP && si == k);
        p.freq[k] = seeded<T>(b.freq[k], false); p.phase[k] = seeded<T>(b.phase[k], false);
        p.samp[k] = seeded<T>(b.scale_amp[k], false);
    }
    p.R = seeded<T>(b.R, me && sp == WL_SEED_R); p.r = seeded<T>(b.r, false);
    p.shell = seeded<T>(b.shell, false); p.sfreq = seeded<T>(b.scale_freq, false); p.sphase = seeded<T>(b.scale_phase, false);
    p.spin = seeded<T>(b.spin, sp == WL_SEED_SPIN && si == which);
    return p;
}

template <class T>
static void gen_wrap_all(GEngine<T>* E, const GLev& g, T* a, int ncomp)
{
    for (int j = 0; j < E->nd; ++j)
        if (g.per[j]) g_planes<T><<<g_blocks(g.nc / g.S[j] * ncomp), G_NT, 0, E->st>>>(g, a, ncomp, j, 0);
}

template <class T>
static void gen_measure(wl_sim* s, GEngine<T>* E, double t)
{
    const GLev& g = E->lev[0];
    g_measure<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->body, T(t), E->mu0, E->mu1, E->V);
    gen_wrap_all<T>(E, g, E->mu0, E->nd);
    gen_wrap_all<T>(E, g, E->mu1, E->nd * E->nd);
    gen_wrap_all<T>(E, g, E->V, E->nd);
    for (int j = 0; j < E->nd; ++j)
        if (!g.per[j]) g_planes<T><<<g_blocks(g.nc / g.S[j]), G_NT, 0, E->st>>>(g, E->mu0 + j * g.nc, 1, j, 1);
    g_diag<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->L[0], E->iD[0]);
    for (int l = 1; l < E->nlev; ++l) {
        g_restrict_L<T><<<g_blocks(E->lev[l].nc), G_NT, 0, E->st>>>(E->lev[l - 1], E->lev[l], E->L[l - 1], E->L[l]);
        g_diag<T><<<g_blocks(E->lev[l].nc), G_NT, 0, E->st>>>(E->lev[l], E->L[l], E->iD[l]);
    }
    s->launches += 4 + 2 * E->nlev;
}

template <class T>
static void gen_bc(wl_sim* s, GEngine<T>* E, T* u)
{
    const GLev& g = E->lev[0];
    for (int j = 0; j < E->nd; ++j) g_bc<T><<<g_blocks(g.nc / g.S[j] * E->nd), G_NT, 0, E->st>>>(g, u, j, E->U[j], E->exit_bc);
    s->launches += E->nd;
}

template <class T>
static void gen_smooth(wl_sim* s, GEngine<T>* E, int l, int its)
{
    const GLev& g = E->lev[l];
    const int nb = G_NB;
    g_pcg_mean_a<T><<<nb, G_NT, 0, E->st>>>(g, E->rr[l], E->iD[l], E->partial);
    g_pcg_mean_b<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc);
    g_pcg_init<T><<<nb, G_NT, 0, E->st>>>(g, E->rr[l], E->iD[l], E->e[l], E->sc, E->partial);
    g_pcg_rho0<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc, E->flags);
    for (int k = 1; k <= its; ++k) {
        g_matvec<T><<<nb, G_NT, 0, E->st>>>(g, E->L[l], E->e[l], E->q[l], E->flags, E->partial);
        g_pcg_alpha<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc, E->flags);
        g_pcg_update<T><<<nb, G_NT, 0, E->st>>>(g, E->x[l], E->rr[l], E->e[l], E->q[l], E->iD[l], E->sc, E->flags, E->partial);
        if (k == its) break;
        g_pcg_beta<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc, E->flags);
        g_pcg_dir<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->e[l], E->rr[l], E->iD[l], E->sc, E->flags);
    }
    s->launches += 4 + 5 * its - 2;
}

template <class T>
static void gen_vcycle(wl_sim* s, GEngine<T>* E, int l)
{
    if (l + 1 >= E->nlev) return;
    const GLev &gf = E->lev[l], &gc = E->lev[l + 1];
    g_restrict_r<T><<<g_blocks(gc.nc), G_NT, 0, E->st>>>(gf, gc, E->rr[l], E->rr[l + 1], E->x[l + 1]);
    if (l + 1 < E->nlev - 1) gen_vcycle<T>(s, E, l + 1);
    gen_smooth<T>(s, E, l + 1, s->cfg.mg.smooth_iters);
    g_prolong_a<T><<<g_blocks(gf.nc), G_NT, 0, E->st>>>(gf, gc, E->x[l + 1], E->e[l]);
    g_prolong_b<T><<<g_blocks(gf.nc), G_NT, 0, E->st>>>(gf, E->L[l], E->e[l], E->x[l], E->rr[l]);
    s->launches += 3;
}

template <class T>
static int gen_project(wl_sim* s, GEngine<T>* E, double w, double dt)
{
    const GLev& g = E->lev[0];
    const wl_mg& mg = s->cfg.mg;
    const T scl = T(w * dt);
    g_div_scale<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->u, E->p, scl, E->sig, E->x[0]);
    g_residual<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->L[0], E->x[0], E->sig, E->rr[0]);
    int nv = 0;
    double res = -1.0;
    if (mg.fixed_vcycles > 0) {
        for (; nv < mg.fixed_vcycles; ++nv) { gen_vcycle<T>(s, E, 0); gen_smooth<T>(s, E, 0, mg.smooth_iters); }
    } else {
        for (;;) {
            g_resmax_a<T><<<G_NB, G_NT, 0, E->st>>>(g, E->rr[0], E->partial);
            g_max_b<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc, GS_RES);
            cudaMemcpyAsync(&E->hsc[GS_RES], &E->sc[GS_RES], sizeof(T), cudaMemcpyDeviceToHost, E->st);
            if (cudaStreamSynchronize(E->st) != cudaSuccess) return WL_ECUDA;
            res = g_val(E->hsc[GS_RES]);
            if (!(res > (double)mg.tol) || nv >= mg.max_vcycles) break;
            gen_vcycle<T>(s, E, 0);
            gen_smooth<T>(s, E, 0, mg.smooth_iters);
            ++nv;
        }
        if (res > (double)mg.tol) { s->noconv = 1; s->noconv_total++; }
    }
    s->vcycles[s->solve_slot] = nv;
    s->res[s->solve_slot] = res;
    g_gradient<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->u, E->L[0], E->x[0], E->p, scl);
    s->launches += 3;
    return WL_OK;
}

template <class T>
static int gen_mom_step(wl_sim* s, GEngine<T>* E, double dt)
{
    const GLev& g = E->lev[0];
    const int nb = g_blocks(g.nc);
    cudaMemcpyAsync(E->u0, E->u, sizeof(T) * g.nc * E->nd, cudaMemcpyDeviceToDevice, E->st);
    for (int stage = 0; stage < 2; ++stage) {
        g_convdiff_f<T><<<nb, G_NT, 0, E->st>>>(g, stage == 0 ? E->u0 : E->u, E->u0, E->V, E->nu, T(dt), E->f);
        gen_wrap_all<T>(E, g, E->f, E->nd);
        g_bdim<T><<<nb, G_NT, 0, E->st>>>(g, E->f, E->V, E->mu0, E->mu1, E->u, stage);
        gen_bc<T>(s, E, E->u);
        if (stage == 0 && E->exit_bc) {
            const int nbe = g_blocks((long long)g.n[1] * g.n[2]) < G_NB ? g_blocks((long long)g.n[1] * g.n[2]) : G_NB;
            cudaMemsetAsync(E->partial, 0, sizeof(double) * 8 * G_NB, E->st);
            g_exit_a<T><<<nbe, G_NT, 0, E->st>>>(g, E->u, E->u0, E->U[0], T(dt), E->partial);
            g_exit_b<T><<<1, G_NT, 0, E->st>>>(g, E->partial, E->U[0], E->sc);
            g_exit_c<T><<<nbe, G_NT, 0, E->st>>>(g, E->u, E->sc);
        }
        s->solve_slot = stage;
        int rc = gen_project<T>(s, E, stage == 0 ? 1.0 : 0.5, dt);
        if (rc != WL_OK) return rc;
        gen_bc<T>(s, E, E->u);
        s->launches += 6;
    }
    return WL_OK;
}

template <class T>
static int gen_create(wl_sim* s, void* ws)
{
    GEngine<T>* E = new (std::nothrow) GEngine<T>();
    if (!E) return WL_ENOMEM;
    memset((void*)E, 0, sizeof(*E));
    const wl_config* c = &s->cfg;
    E->st = s->st;
    const size_t need = gen_layout<T>(E, c, ws);
    if (cudaMemsetAsync(ws, 0, need, E->st) != cudaSuccess) { delete E; return WL_ECUDA; }
    if (cudaMallocHost((void**)&E->hsc, sizeof(T) * GS_COUNT + sizeof(int) * GF_COUNT) != cudaSuccess) { delete E; return WL_ECUDA; }
    E->hflags = (int*)(E->hsc + GS_COUNT);
    memset((void*)E->hsc, 0, sizeof(T) * GS_COUNT + sizeof(int) * GF_COUNT);
    const int sp = c->tangent_param;
    E->nu = seeded<T>(c->nu, sp == WL_SEED_NU);
    for (int k = 0; k < 3; ++k) E->U[k] = seeded<T>(c->U[k], sp == WL_SEED_U && c->tangent_index == k);
    E->eps = seeded<T>(c->eps, false);
    E->exit_bc = c->exit_bc;
    E->body.n = c->body.kind == WL_BODY_NONE ? 0 : 1 + c->nextra;
    E->body.eps = E->eps;
    for (int e = 0; e < E->body.n; ++e) E->body.part[e] = make_part<T>(e == 0 ? c->body : c->extra[e - 1], e == 0 ? 0 : c->extra_op[e - 1], c, e);
    s->gen = E;
    s->nd = E->nd; s->nlev = E->nlev;
    // initial state (R-V): u = U everywhere, p = 0, measure(0), BC fill
    const GLev& g = E->lev[0];
    for (int i = 0; i < E->nd; ++i) g_fill<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(E->u + i * g.nc, g.nc, E->U[i]);
    cudaMemcpyAsync(E->u0, E->u, sizeof(T) * g.nc * E->nd, cudaMemcpyDeviceToDevice, E->st);
    gen_measure<T>(s, E, 0.0);
    gen_bc<T>(s, E, E->u);
    if (cudaStreamSynchronize(E->st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { cudaFreeHost(E->hsc); delete E; s->gen = nullptr; return WL_ECUDA; }
    return WL_OK;
}

template <class T>
static T* gen_find(GEngine<T>* E, const char* name, int level, int* ncomp, const GLev** g)
{
    *ncomp = 1;
    if (level < 0 || level >= E->nlev) return nullptr;
    *g = &E->lev[level];
    if (!strcmp(name, "L")) { *ncomp = E->nd; return E->L[level]; }
    if (!strcmp(name, "iD")) return E->iD[level];
    if (!strcmp(name, "x")) return E->x[level];
    if (!strcmp(name, "r")) return E->rr[level];
    *g = &E->lev[0];
    if (!strcmp(name, "u")) { *ncomp = E->nd; return E->u; }
    if (!strcmp(name, "p")) return E->p;
    if (!strcmp(name, "mu0")) { *ncomp = E->nd; return E->mu0; }
    if (!strcmp(name, "mu1")) { *ncomp = E->nd * E->nd; return E->mu1; }
    if (!strcmp(name, "V")) { *ncomp = E->nd; return E->V; }
    return nullptr;
}

// interior copy of `ncomp` arrays to a user buffer of F (host or device), lane 0 value / 1 derivative; staging in E->f / E->sig
template <class T, class F>
static int gen_copy_out(wl_sim* s, GEngine<T>* E, const GLev& g, const T* a, int ncomp, F* dst, int on_device, int lane)
{
    const long long ni = (long long)g.n[0] * g.n[1] * g.n[2];
    for (int m = 0; m < ncomp; ++m) {
        F* stage = on_device ? dst + m * ni : (F*)E->q[0];       // q of level 0 is scratch between solves (>= ni doubles)
        g_pack<T, F><<<g_blocks(ni), G_NT, 0, E->st>>>(g, a + m * g.nc, stage, 1, lane);
        if (!on_device) {
            if (cudaMemcpyAsync(dst + m * ni, stage, sizeof(F) * ni, cudaMemcpyDeviceToHost, E->st) != cudaSuccess) return WL_ECUDA;
            if (cudaStreamSynchronize(E->st) != cudaSuccess) return WL_ECUDA;
        }
    }
    s->launches += ncomp;
    return cudaGetLastError() == cudaSuccess ? WL_OK : WL_ECUDA;
}
template <class T, class F>
static int gen_copy_in(wl_sim* s, GEngine<T>* E, const GLev& g, T* a, int ncomp, const F* src, int on_device)
{
    const long long ni = (long long)g.n[0] * g.n[1] * g.n[2];
    for (int m = 0; m < ncomp; ++m) {
        const F* stage = src + m * ni;
        if (!on_device) {
            if (cudaMemcpyAsync(E->q[0], src + m * ni, sizeof(F) * ni, cudaMemcpyHostToDevice, E->st) != cudaSuccess) return WL_ECUDA;
            stage = (const F*)E->q[0];
        }
        g_unpack<T, F><<<g_blocks(ni), G_NT, 0, E->st>>>(g, stage, a + m * g.nc, 1);
        if (!on_device && cudaStreamSynchronize(E->st) != cudaSuccess) return WL_ECUDA;
    }
    s->launches += ncomp;
    return cudaGetLastError() == cudaSuccess ? WL_OK : WL_ECUDA;
}

// ---- dispatch over the two instantiations
#define GEN_CALL(s, EXPR_D, EXPR_T) ((s)->gen_kind == 1 ? (EXPR_D) : (EXPR_T))
#define ED(s) ((GEngine<double>*)(s)->gen)
#define ET(s) ((GEngine<Dual>*)(s)->gen)

size_t wl_gen_bytes(const wl_config* c)
{
    return c->tangent_param != WL_SEED_NONE ? gen_layout<Dual>(nullptr, c, nullptr) : gen_layout<double>(nullptr, c, nullptr);
}
int wl_gen_create(wl_sim* s, void* ws)
{
    s->gen_kind = s->cfg.tangent_param != WL_SEED_NONE ? 2 : 1;
    return s->gen_kind == 1 ? gen_create<double>(s, ws) : gen_create<Dual>(s, ws);
}
void wl_gen_destroy(wl_sim* s)
{
    if (!s->gen) return;
    if (s->gen_kind == 1) { cudaFreeHost(ED(s)->hsc); delete ED(s); } else { cudaFreeHost(ET(s)->hsc); delete ET(s); }
    s->gen = nullptr;
}
int wl_gen_measure(wl_sim* s, double t)
{
    if (s->gen_kind == 1) gen_measure<double>(s, ED(s), t); else gen_measure<Dual>(s, ET(s), t);
    return cudaGetLastError() == cudaSuccess ? WL_OK : WL_ECUDA;
}
int wl_gen_mom_step(wl_sim* s, double dt)
{
    int rc = GEN_CALL(s, gen_mom_step<double>(s, ED(s), dt), gen_mom_step<Dual>(s, ET(s), dt));
    if (rc != WL_OK) return rc;
    return cudaGetLastError() == cudaSuccess ? WL_OK : WL_ECUDA;
}
template <class T>
static int gen_cfl(wl_sim* s, GEngine<T>* E, float* dt_out)
{
    const GLev& g = E->lev[0];
    cudaMemsetAsync(&E->flags[GF_NAN], 0, sizeof(int), E->st);
    g_cfl_a<T><<<G_NB, G_NT, 0, E->st>>>(g, E->u, E->partial, E->flags);
    g_max_b<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc, GS_CFL);
    cudaMemcpyAsync(&E->hsc[GS_CFL], &E->sc[GS_CFL], sizeof(T), cudaMemcpyDeviceToHost, E->st);
    cudaMemcpyAsync(E->hflags, E->flags, sizeof(int) * GF_COUNT, cudaMemcpyDeviceToHost, E->st);
    if (cudaStreamSynchronize(E->st) != cudaSuccess) return WL_ECUDA;
    const wl_config& c = s->cfg;
    const double dt = (double)c.cfl_c / (g_val(E->hsc[GS_CFL]) + (double)c.cfl_cnu * (double)c.nu);
    *dt_out = (float)(dt < (double)c.dt_max ? dt : (double)c.dt_max);
    s->hs->nan_flag = E->hflags[GF_NAN];
    s->launches += 2;
    return WL_OK;
}
int wl_gen_cfl(wl_sim* s, float* dt_out) { return GEN_CALL(s, gen_cfl<double>(s, ED(s), dt_out), gen_cfl<Dual>(s, ET(s), dt_out)); }

template <class T>
static int gen_reduce3(wl_sim* s, GEngine<T>* E, int slot, int nv, double* out, double* dout)
{
    g_sum_b<T><<<1, G_NT, 0, E->st>>>(E->partial, E->sc, slot, nv);
    cudaMemcpyAsync(&E->hsc[slot], &E->sc[slot], sizeof(T) * nv, cudaMemcpyDeviceToHost, E->st);
    if (cudaStreamSynchronize(E->st) != cudaSuccess) return WL_ECUDA;
    for (int k = 0; k < nv; ++k) { out[k] = g_val(E->hsc[slot + k]); if (dout) dout[k] = g_der(E->hsc[slot + k]); }
    s->launches += 2;
    return WL_OK;
}
template <class T>
static int gen_force(wl_sim* s, GEngine<T>* E, double t, double* F, double* dF)
{
    g_force_a<T><<<G_NB, G_NT, 0, E->st>>>(E->lev[0], E->body, T(t), E->p, E->partial);
    return gen_reduce3<T>(s, E, GS_F0, 3, F, dF);
}
int wl_gen_force(wl_sim* s, double t, double* F, double* dF) { return GEN_CALL(s, gen_force<double>(s, ED(s), t, F, dF), gen_force<Dual>(s, ET(s), t, F, dF)); }
template <class T>
static int gen_energy(wl_sim* s, GEngine<T>* E, double* out, double* dout)
{
    g_energy_a<T><<<G_NB, G_NT, 0, E->st>>>(E->lev[0], E->u, E->partial);
    return gen_reduce3<T>(s, E, GS_KE, 2, out, dout);
}
int wl_gen_energy(wl_sim* s, double* out, double* dout) { return GEN_CALL(s, gen_energy<double>(s, ED(s), out, dout), gen_energy<Dual>(s, ET(s), out, dout)); }

template <class T>
static int gen_init_tgv(wl_sim* s, GEngine<T>* E, int sign)
{
    const GLev& g = E->lev[0];
    g_init_tgv<T><<<g_blocks(g.nc), G_NT, 0, E->st>>>(g, E->u, E->p, sign);
    gen_bc<T>(s, E, E->u);
    return cudaGetLastError() == cudaSuccess ? WL_OK : WL_ECUDA;
}
int wl_gen_init_tgv(wl_sim* s, int sign) { return GEN_CALL(s, gen_init_tgv<double>(s, ED(s), sign), gen_init_tgv<Dual>(s, ET(s), sign)); }

template <class T, class F>
static int gen_set(wl_sim* s, GEngine<T>* E, const F* u, const F* p, int on_device)
{
    int rc;
    if (u) { if ((rc = gen_copy_in<T, F>(s, E, E->lev[0], E->u, E->nd, u, on_device)) != WL_OK) return rc; gen_bc<T>(s, E, E->u); }
    if (p && (rc = gen_copy_in<T, F>(s, E, E->lev[0], E->p, 1, p, on_device)) != WL_OK) return rc;
    return cudaStreamSynchronize(E->st) == cudaSuccess ? WL_OK : WL_ECUDA;
}
int wl_gen_set_fields(wl_sim* s, const float* u, const float* p, int on_device)
{
    return GEN_CALL(s, (gen_set<double, float>(s, ED(s), u, p, on_device)), (gen_set<Dual, float>(s, ET(s), u, p, on_device)));
}
int wl_gen_set_fields_f64(wl_sim* s, const double* u, const double* p, int on_device)
{
    return GEN_CALL(s, (gen_set<double, double>(s, ED(s), u, p, on_device)), (gen_set<Dual, double>(s, ET(s), u, p, on_device)));
}
template <class T, class F>
static int gen_get(wl_sim* s, GEngine<T>* E, F* u, F* p, F* mu0, int on_device, int lane)
{
    int rc;
    if (u && (rc = gen_copy_out<T, F>(s, E, E->lev[0], E->u, E->nd, u, on_device, lane)) != WL_OK) return rc;
    if (p && (rc = gen_copy_out<T, F>(s, E, E->lev[0], E->p, 1, p, on_device, lane)) != WL_OK) return rc;
    if (mu0 && (rc = gen_copy_out<T, F>(s, E, E->lev[0], E->mu0, E->nd, mu0, on_device, lane)) != WL_OK) return rc;
    return cudaStreamSynchronize(E->st) == cudaSuccess ? WL_OK : WL_ECUDA;
}
int wl_gen_get_fields(wl_sim* s, float* u, float* p, float* mu0, int on_device)
{
    return GEN_CALL(s, (gen_get<double, float>(s, ED(s), u, p, mu0, on_device, 0)), (gen_get<Dual, float>(s, ET(s), u, p, mu0, on_device, 0)));
}
int wl_gen_get_fields_f64(wl_sim* s, double* u, double* p, int lane, int on_device)
{
    if (lane == 1 && s->gen_kind != 2) return WL_EINVAL;
    return GEN_CALL(s, (gen_get<double, double>(s, ED(s), u, p, nullptr, on_device, 0)), (gen_get<Dual, double>(s, ET(s), u, p, nullptr, on_device, lane)));
}
template <class T>
static int gen_dbg_get(wl_sim* s, GEngine<T>* E, const char* name, int level, int lane, double* out, size_t n)
{
    int nc; const GLev* g = nullptr;
    T* a = gen_find<T>(E, name, level, &nc, &g);
    if (!a) return WL_EINVAL;
    const size_t ni = (size_t)g->n[0] * g->n[1] * g->n[2];
    if (n < ni * nc) return WL_EINVAL;
    int rc = gen_copy_out<T, double>(s, E, *g, a, nc, out, 0, lane);
    return rc != WL_OK ? rc : nc;
}
int wl_gen_dbg_get(wl_sim* s, const char* name, int level, int lane, double* out, size_t n)
{
    if (lane == 1 && s->gen_kind != 2) return WL_EINVAL;
    return GEN_CALL(s, gen_dbg_get<double>(s, ED(s), name, level, lane, out, n), gen_dbg_get<Dual>(s, ET(s), name, level, lane, out, n));
}
