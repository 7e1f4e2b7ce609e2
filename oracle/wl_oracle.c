/*
 * wl_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for one time step (mom_step) of the incompressible
 * BDIM flow solver described in arXiv 2407.16032 (PAPER.md, cited "P:<line>").
 * It shares no code with the CUDA path (paper_2407_16032_b200/csrc) and neither imports
 * the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * The paper names its numerical steps but defers every formula to cited works
 * (P:74-76).  Each function below therefore follows the *reading* written down in
 * DESIGN.md section 3 ("R-<x>"), which restates SURVEY.md section 8(c) items O1..O11; the
 * comment on each function names the passage of the paper and the reading it follows.
 *
 * Indexing.  Paper arrays are 1-based with one ghost cell per side, interior
 * I_d = 2..N_d+1 (size 10 -> inside = 2:9).  Here arrays are 0-based C arrays of
 * padded size S_d = N_d+2, so C index c_d = I_d - 1: interior c_d = 1..N_d, ghosts 0
 * and N_d+1.  x is fastest.  Unit grid spacing h = 1 ("all grid cells are
 * identical, no grid information is stored").  Cell c has centre x_c = c - 1/2, the
 * domain is [0,N_d]; u_i[c] lives on the LOWER i-face of cell c, at x_c - e_i/2, which
 * is what the pressure-gradient kernel u[I,i] -= c[I,i]*(p[I]-p[I-d(i)]) of P:88 forces.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): kernel moments vs quadrature,
 * SDF gradients vs finite differences, body volume, conv_diff invariants and
 * convergence order, Laplacian special case vs a textbook kron Laplacian, operator
 * symmetry / null space, multigrid vs dense direct solve on 16x16, divergence after
 * projection, free-stream preservation, 2-D Taylor-Green closed-form decay, CFL closed
 * forms, force vs divergence theorem; the two constants the readings add (the decoupling
 * threshold of level_diag, the relative stop of wlo_smooth) by hand-set coefficients and by a
 * two-eigenmode residual with closed-form iterates; general bodies (shell, non-rigid map, spin, SDF arithmetic) by the
 * uniformly scaled sphere, finite differences of the map, and the paper's jellyfish listing.  No function here is "parity unpinned" except
 * whole-run physical values (C_D etc.), which need the paper's run lengths and data.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define WLO_MAXLEV 16
#define WLO_PI 3.14159265358979323846

enum { WLO_BODY_NONE = 0, WLO_BODY_SPHERE = 1, WLO_BODY_TORUS = 2, WLO_BODY_CYLINDER = 3, WLO_BODY_PLANE = 4 };
enum { WLO_OP_UNION = 0, WLO_OP_DIFFERENCE = 1 };
#define WLO_MAX_EXTRA 3
enum { WLO_MOTION_STATIC = 0, WLO_MOTION_SIN = 1 };

/* one further primitive of a composite body (SDF arithmetic, "body = big + small", "sphere - plane"):
 * the same fields as the first primitive, which lives in wlo_config itself */
typedef struct {
    int kind;
    double centre[3];
    double R, r;
    int axis;
    int motion;
    double amp[3], freq[3], phase[3];
    double shell;
    double scale_amp[3], scale_freq, scale_phase;
    double spin;
    int op;             /* WLO_OP_*: how this primitive combines with the body built so far */
} wlo_part;

typedef struct {
    int ndim;
    int dims[3];        /* interior cells N_d */
    double L;           /* length scale (only scales reported quantities) */
    double U[3];        /* boundary / inflow velocity */
    double nu;          /* viscosity in grid units */
    int periodic[3];
    int exit_bc;        /* convective exit on the +x plane */
    double eps;         /* BDIM kernel half-width (cells) */
    double dt0, dt_max, cfl_c, cfl_cnu;
    /* body: SDF + translation map */
    int body_kind;
    double centre[3];
    double R, r;        /* sphere / cylinder radius R; torus major R, minor r */
    int axis;           /* torus / cylinder axis */
    int motion;
    double amp[3], freq[3], phase[3];   /* c_d(t) = centre[d] + amp[d] sin(2 pi freq[d] t + phase[d]) */
    /* multigrid */
    int max_levels, smooth_iters, max_vcycles, fixed_vcycles;
    double tol;
    /* general bodies (reading R-E3): thin shell, non-rigid diagonal map, spin, further primitives */
    double shell;       /* > 0: the body is the shell of this half-thickness around the surface: sdf <- |sdf| - shell */
    double scale_amp[3], scale_freq, scale_phase;   /* map xi_d = s_d(t) (x_d - c_d(t)), s_d = 1 + scale_amp[d] cos(2 pi scale_freq t + scale_phase) ("A(t) .* x + B(t)") */
    double spin;        /* angular velocity of the primitive about its axis (z in 2-D) through its centre: the SDF is unchanged
                           (bodies of revolution about that axis), the surface velocity is not ("spinning circles") */
    int nextra;
    wlo_part extra[WLO_MAX_EXTRA];
} wlo_config;

typedef struct {
    int n[3];           /* interior cells */
    int S[3];           /* padded sizes */
    long st[3];         /* strides */
    long ncell;         /* padded cell count */
    double *L;          /* nd face coefficients (level 0: alias of mu0) */
    double *iD, *x, *r, *e, *q;
} wlo_level;

typedef struct wlo_sim {
    wlo_config cfg;
    int nd, nlev;
    wlo_level lev[WLO_MAXLEV];
    double *u, *u0, *f, *p, *sig, *V, *mu0, *mu1;
    int last_vcycles[2];
    double last_res[2];
    int solve_slot;
} wlo_sim;

/* ------------------------------------------------------------------ helpers */

static inline long IDX(const wlo_level *g, int c0, int c1, int c2)
{
    return c0 * g->st[0] + c1 * g->st[1] + c2 * g->st[2];
}

/* wrap a padded index into the interior 1..N in a periodic direction; otherwise leave
 * it (it then addresses a ghost cell). */
static inline int wrapc(int c, int N, int per)
{
    if (per) {
        if (c < 1) c += N;
        else if (c > N) c -= N;
    }
    return c;
}

static void level_alloc(wlo_level *g, int nd, const int *n, int own_L)
{
    long nc = 1;
    for (int d = 0; d < 3; ++d) {
        g->n[d] = d < nd ? n[d] : 1;
        g->S[d] = d < nd ? n[d] + 2 : 1;
    }
    g->st[0] = 1; g->st[1] = g->S[0]; g->st[2] = (long)g->S[0] * g->S[1];
    if (nd < 3) g->st[2] = 0;
    nc = (long)g->S[0] * g->S[1] * g->S[2];
    g->ncell = nc;
    g->L = own_L ? (double *)calloc((size_t)nc * nd, sizeof(double)) : NULL;
    g->iD = (double *)calloc((size_t)nc, sizeof(double));
    g->x = (double *)calloc((size_t)nc, sizeof(double));
    g->r = (double *)calloc((size_t)nc, sizeof(double));
    g->e = (double *)calloc((size_t)nc, sizeof(double));
    g->q = (double *)calloc((size_t)nc, sizeof(double));
}

/* loop bounds: interior in every direction; in 2-D the z loop runs once at c2 = 0 */
#define ZLO(g, nd) ((nd) == 3 ? 1 : 0)
#define ZHI(g, nd) ((nd) == 3 ? (g)->n[2] : 0)

/* -------------------------------------------------- O1: BDIM kernel moments
 * P:70-72 "immersed-boundary thickness eps defines the region ..." gives no kernel;
 * reading R-B: cosine kernel K(s) = (1+cos(pi s/eps))/(2 eps), |s|<eps.
 *   mu0(d) = int_{-eps}^{d} K ds,   mu1(d) = int_{-d}^{eps} s K ds,   d clamped to [-eps,eps].
 */
double wlo_kernel_K(double s, double eps)
{
    if (fabs(s) >= eps) return 0.0;
    return (1.0 + cos(WLO_PI * s / eps)) / (2.0 * eps);
}
double wlo_kernel_mu0(double d, double eps)
{
    double a = d / eps;
    if (a <= -1.0) return 0.0;
    if (a >= 1.0) return 1.0;
    return 0.5 + 0.5 * a + sin(WLO_PI * a) / (2.0 * WLO_PI);
}
double wlo_kernel_mu1(double d, double eps)
{
    double a = d / eps;
    if (a <= -1.0 || a >= 1.0) return 0.0;
    return eps * (0.25 - 0.25 * a * a
                  - (a * sin(WLO_PI * a) + (1.0 + cos(WLO_PI * a)) / WLO_PI) / (2.0 * WLO_PI));
}

/* -------------------------------------------------- O2: body SDF, normal, velocity
 * P:104 "AutoBody type holds the signed-distance function as well as the coordinates
 * mapping"; "signed-distance d and normal n from any point in space".  Reading R-E:
 * analytic gradients of the parametric SDFs (same values the paper gets by AD).
 * Reading R-E3 (general bodies, SURVEY O2 "n = J^T grad sdf / |.|, V = -J^-1 dmap/dt"):
 *   map     xi_d = s_d(t) (x_d - c_d(t)),  c_d(t) = c0_d + amp_d sin(2 pi f_d t + phase_d)   (translation; the heaving
 *           sphere of BASELINE configs[4]: one direction; the 2-DOF cylinder of P:181: two),
 *           s_d(t) = 1 + scale_amp_d cos(2 pi scale_freq t + scale_phase)                    (the "A(t) .* x" of P:237);
 *           J = diag(s).
 *   sdf     d0 = sdf(xi) of the primitive, g = grad_xi sdf; shell > 0: d0 <- |d0| - shell, g <- sign(d0) g;
 *   normal  grad_x d0 = J^T g = s .* g, m = |s .* g|; n = (s .* g)/m;
 *   distance d = d0/m: the first-order distance in physical space (exact for a uniformly scaled sphere: |x-c| - R/s);
 *           m < 1e-12 => n = 0, d = d0; a rigid map (every scale_amp = 0) skips the normalisation: d = d0, n = g as in R-E;
 *   velocity a material point has fixed xi: x(t) = c + xi ./ s, so V_d = dc_d/dt - (ds_d/dt / s_d)(x_d - c_d)  (= -J^-1 dmap/dt),
 *           plus spin * e_axis x (x - c) for a primitive spinning about its axis.
 * Primitives: sphere |xi| - R (circle in 2-D); torus (axis a); circular cylinder of P:121 (radius R, axis e_a, spanning a
 * periodic direction) rho - R; half-space xi_a (below the plane through the centre with normal +e_a).
 * SDF arithmetic: union  d = min(d_A, d_B), difference A - B  d = max(d_A, -d_B); normal and velocity are
 * those of the primitive that decides (for -d_B: -n_B, V_B).
 * Returns d; fills nrm[3], vel[3].
 */
static double prim_sdf(int nd, int kind, int axis, double R, double r, const double *xi, double *g)
{
    g[0] = g[1] = g[2] = 0.0;
    if (kind == WLO_BODY_SPHERE) {               /* circle in 2-D */
        double rr = 0;
        for (int k = 0; k < nd; ++k) rr += xi[k] * xi[k];
        rr = sqrt(rr);
        if (rr >= 1e-12) for (int k = 0; k < nd; ++k) g[k] = xi[k] / rr;
        return rr - R;
    }
    if (kind == WLO_BODY_PLANE) { g[axis] = 1.0; return xi[axis]; }
    /* torus and cylinder (3-D): axis a; rho = distance from the axis in the (b,c) plane */
    int a = axis, b = (a + 1) % 3, cc = (a + 2) % 3;
    double rho = sqrt(xi[b] * xi[b] + xi[cc] * xi[cc]);
    if (kind == WLO_BODY_CYLINDER) {
        if (rho >= 1e-12) { g[b] = xi[b] / rho; g[cc] = xi[cc] / rho; }
        return rho - R;
    }
    double w = rho - R;
    double q = sqrt(w * w + xi[a] * xi[a]);
    if (q >= 1e-12 && rho >= 1e-12) {
        g[a] = xi[a] / q;
        g[b] = (w / q) * (xi[b] / rho);
        g[cc] = (w / q) * (xi[cc] / rho);
    } else if (q >= 1e-12) {
        g[a] = xi[a] / q;       /* on the axis: in-plane direction undefined */
    }
    return q - r;
}

static double part_eval(int nd, const wlo_part *p, const double *xpt, double t, double *nrm, double *vel)
{
    double c[3], cdot[3] = { 0, 0, 0 }, sc[3] = { 1, 1, 1 }, sdot[3] = { 0, 0, 0 }, xi[3] = { 0, 0, 0 }, g[3];
    for (int k = 0; k < 3; ++k) c[k] = p->centre[k];
    if (p->motion == WLO_MOTION_SIN)
        for (int k = 0; k < nd; ++k) {
            double ph = 2.0 * WLO_PI * p->freq[k] * t + p->phase[k];
            c[k] += p->amp[k] * sin(ph);
            cdot[k] = p->amp[k] * 2.0 * WLO_PI * p->freq[k] * cos(ph);
        }
    {
        double ph = 2.0 * WLO_PI * p->scale_freq * t + p->scale_phase;
        for (int k = 0; k < nd; ++k) {
            sc[k] = 1.0 + p->scale_amp[k] * cos(ph);
            sdot[k] = -p->scale_amp[k] * 2.0 * WLO_PI * p->scale_freq * sin(ph);
        }
    }
    for (int k = 0; k < nd; ++k) xi[k] = sc[k] * (xpt[k] - c[k]);
    double d0 = prim_sdf(nd, p->kind, p->axis, p->R, p->r, xi, g);
    if (p->shell > 0.0) {
        double sg = d0 < 0.0 ? -1.0 : 1.0;
        d0 = fabs(d0) - p->shell;
        for (int k = 0; k < 3; ++k) g[k] *= sg;
    }
    nrm[0] = nrm[1] = nrm[2] = 0.0;
    double d = d0;
    if (p->scale_amp[0] == 0.0 && p->scale_amp[1] == 0.0 && p->scale_amp[2] == 0.0) {
        for (int k = 0; k < nd; ++k) nrm[k] = g[k];          /* rigid map: the SDF is exact, g is the unit normal (R-E) */
    } else {
        double m = 0;
        for (int k = 0; k < nd; ++k) { g[k] *= sc[k]; m += g[k] * g[k]; }
        m = sqrt(m);
        if (m >= 1e-12) {
            d = d0 / m;
            for (int k = 0; k < nd; ++k) nrm[k] = g[k] / m;
        }
    }
    vel[0] = vel[1] = vel[2] = 0.0;
    for (int k = 0; k < nd; ++k) vel[k] = cdot[k] - (sdot[k] / sc[k]) * (xpt[k] - c[k]);
    if (p->spin != 0.0) {                        /* spin e_a x (x - c); 2-D: a = z */
        int a = nd == 3 ? p->axis : 2, b = (a + 1) % 3, cc = (a + 2) % 3;
        double xb = b < nd ? xpt[b] - c[b] : 0.0, xc = cc < nd ? xpt[cc] - c[cc] : 0.0;
        if (b < nd) vel[b] += -p->spin * xc;
        if (cc < nd) vel[cc] += p->spin * xb;
    }
    return d;
}

double wlo_body_eval(const wlo_config *cf, const double *xpt, double t, double *nrm, double *vel)
{
    int nd = cf->ndim;
    nrm[0] = nrm[1] = nrm[2] = 0.0;
    vel[0] = vel[1] = vel[2] = 0.0;
    if (cf->body_kind == WLO_BODY_NONE) return 1e30;
    wlo_part first;
    memset(&first, 0, sizeof(first));
    first.kind = cf->body_kind; first.R = cf->R; first.r = cf->r; first.axis = cf->axis; first.motion = cf->motion;
    first.shell = cf->shell; first.scale_freq = cf->scale_freq; first.scale_phase = cf->scale_phase; first.spin = cf->spin;
    for (int k = 0; k < 3; ++k) {
        first.centre[k] = cf->centre[k]; first.amp[k] = cf->amp[k]; first.freq[k] = cf->freq[k]; first.phase[k] = cf->phase[k];
        first.scale_amp[k] = cf->scale_amp[k];
    }
    double d = part_eval(nd, &first, xpt, t, nrm, vel);
    for (int e = 0; e < cf->nextra; ++e) {
        double n2[3], v2[3];
        double d2 = part_eval(nd, &cf->extra[e], xpt, t, n2, v2);
        if (cf->extra[e].op == WLO_OP_DIFFERENCE) {
            d2 = -d2;
            for (int k = 0; k < 3; ++k) n2[k] = -n2[k];
            if (d2 > d) { d = d2; for (int k = 0; k < 3; ++k) { nrm[k] = n2[k]; vel[k] = v2[k]; } }
        } else if (d2 < d) {
            d = d2;
            for (int k = 0; k < 3; ++k) { nrm[k] = n2[k]; vel[k] = v2[k]; }
        }
    }
    return d;
}

/* -------------------------------------------------- O7: Poisson diagonal
 * D_I = -sum_i (L[I,i] + L[I+d_i,i]);  iD = 1/D if |D| > 2n*1e-6 else 0 (reading R-O/S:
 * cells buried in the body decouple).  The threshold (WLO_DMIN per face) instead of an exact
 * test for zero keeps cells whose faces all sit within ~1e-2 eps of the d = -eps shell out
 * of the solve: their mu0 ~ 1e-6 or less, so 1/D would multiply fp32 round-off in div u by
 * 1e6 or more and dominate the CG dot products.
 */
#define WLO_DMIN 1e-6
static void level_diag(wlo_level *g, int nd)
{
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                double D = 0;
                for (int i = 0; i < nd; ++i)
                    D -= g->L[i * g->ncell + id] + g->L[i * g->ncell + id + g->st[i]];
                g->iD[id] = fabs(D) > 2.0 * nd * WLO_DMIN ? 1.0 / D : 0.0;
            }
}

/* fill the ghosts of a scalar level array by periodic wrap (periodic directions only) */
static void level_wrap(const wlo_sim *s, const wlo_level *g, double *a)
{
    int nd = s->nd;
    for (int j = 0; j < nd; ++j) {
        if (!s->cfg.periodic[j]) continue;
        int N = g->n[j];
        int lo[3] = { 0, 0, 0 }, hi[3] = { g->S[0] - 1, g->S[1] - 1, g->S[2] - 1 };
        lo[j] = hi[j] = 0;
        for (int c2 = lo[2]; c2 <= hi[2]; ++c2)
            for (int c1 = lo[1]; c1 <= hi[1]; ++c1)
                for (int c0 = lo[0]; c0 <= hi[0]; ++c0) {
                    long b = IDX(g, c0, c1, c2);        /* c_j = 0 */
                    a[b] = a[b + N * g->st[j]];
                    a[b + (N + 1) * g->st[j]] = a[b + g->st[j]];
                }
    }
}

/* coefficient restriction (reading R-S): coarse face coefficient = 1/2 * sum of the
 * 2^(n-1) fine-face coefficients lying on that coarse face. */
static void restrict_coeffs(const wlo_sim *s, const wlo_level *f, wlo_level *c)
{
    int nd = s->nd;
    for (int i = 0; i < nd; ++i) {
        const double *Lf = f->L + i * f->ncell;
        double *Lc = c->L + i * c->ncell;
        /* faces C_i = 1..n_i+1, other directions interior */
        int hi[3] = { c->n[0], c->n[1], nd == 3 ? c->n[2] : 0 };
        hi[i] += 1;
        for (int C2 = ZLO(c, nd); C2 <= hi[2]; ++C2)
            for (int C1 = 1; C1 <= hi[1]; ++C1)
                for (int C0 = 1; C0 <= hi[0]; ++C0) {
                    int C[3] = { C0, C1, C2 };
                    int b[3];
                    for (int d = 0; d < 3; ++d) b[d] = d < nd ? 2 * C[d] - 1 : 0;
                    double sum = 0;
                    int n1 = (nd >= 2) ? 2 : 1, n2 = (nd == 3) ? 2 : 1;
                    /* iterate the children in the directions other than i */
                    for (int a2 = 0; a2 < n2; ++a2)
                        for (int a1 = 0; a1 < n1; ++a1)
                            for (int a0 = 0; a0 < 2; ++a0) {
                                int a[3] = { a0, a1, a2 };
                                if (a[i] != 0) continue;   /* stay on the face */
                                sum += Lf[IDX(f, b[0] + a[0], b[1] + a[1], b[2] + a[2])];
                            }
                    Lc[IDX(c, C0, C1, C2)] = 0.5 * sum;
                }
    }
}

static void poisson_update(wlo_sim *s)
{
    level_diag(&s->lev[0], s->nd);
    for (int l = 1; l < s->nlev; ++l) {
        restrict_coeffs(s, &s->lev[l - 1], &s->lev[l]);
        level_diag(&s->lev[l], s->nd);
    }
}

/* -------------------------------------------------- O2: measure(t)
 * P:139 "measure!: coordinates mapping for a moving solid boundary".
 * For each face (c,i) of the whole padded array, x_f = x_c(c) - e_i/2:
 *   mu0[c,i] = mu0(d), mu1[c,i,j] = mu1(d) n_j, V[c,i] = V_i.
 * Then the domain rule (reading R-O): non-periodic j => mu0 = 0 on the two boundary-
 * normal faces c_j = 1 and c_j = N_j+1 (homogeneous-Neumann Poisson problem); periodic j
 * => ghosts of mu0, mu1, V wrapped.  Finally the Poisson diagonal and the coarse
 * coefficients are refreshed.
 */
void wlo_measure(wlo_sim *s, double t)
{
    const wlo_config *cf = &s->cfg;
    wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
    double eps = cf->eps;
#pragma omp parallel for collapse(2)
    for (int c2 = 0; c2 < g->S[2]; ++c2)
        for (int c1 = 0; c1 < g->S[1]; ++c1)
            for (int c0 = 0; c0 < g->S[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                int c[3] = { c0, c1, c2 };
                for (int i = 0; i < nd; ++i) {
                    double xf[3], nrm[3], vel[3];
                    for (int k = 0; k < 3; ++k) xf[k] = k < nd ? c[k] - 0.5 : 0.0;
                    xf[i] -= 0.5;
                    double d = wlo_body_eval(cf, xf, t, nrm, vel);
                    double m0 = cf->body_kind == WLO_BODY_NONE ? 1.0 : wlo_kernel_mu0(d, eps);
                    double m1 = cf->body_kind == WLO_BODY_NONE ? 0.0 : wlo_kernel_mu1(d, eps);
                    s->mu0[i * nc + id] = m0;
                    for (int j = 0; j < nd; ++j) s->mu1[(i * nd + j) * nc + id] = m1 * nrm[j];
                    s->V[i * nc + id] = vel[i];
                }
            }
    for (int i = 0; i < nd; ++i) level_wrap(s, g, s->mu0 + i * nc);
    for (int i = 0; i < nd * nd; ++i) level_wrap(s, g, s->mu1 + i * nc);
    for (int i = 0; i < nd; ++i) level_wrap(s, g, s->V + i * nc);
    for (int j = 0; j < nd; ++j) {
        if (cf->periodic[j]) continue;
        double *m = s->mu0 + j * nc;
        int lo[3] = { 0, 0, 0 }, hi[3] = { g->S[0] - 1, g->S[1] - 1, g->S[2] - 1 };
        lo[j] = hi[j] = 0;
        for (int c2 = lo[2]; c2 <= hi[2]; ++c2)
            for (int c1 = lo[1]; c1 <= hi[1]; ++c1)
                for (int c0 = lo[0]; c0 <= hi[0]; ++c0) {
                    long b = IDX(g, c0, c1, c2);
                    m[b + g->st[j]] = 0.0;
                    m[b + (g->n[j] + 1) * g->st[j]] = 0.0;
                }
    }
    poisson_update(s);
}

/* -------------------------------------------------- O5: BC fill
 * P:104 "slip by default, otherwise a convective outlet or a periodic condition".
 * Reading R-M.  For each direction j in order x, y, z (loops span the whole padded range
 * of the other directions, so edges/corners are defined by composition):
 *   periodic:  u[c_j=0] = u[N_j], u[N_j+1] = u[1]       (all components)
 *   otherwise: normal component u_j := U_j at c_j in {0,1} and at c_j = N_j+1
 *              (the upper one is left alone when exit_bc and j = x);
 *              tangential components: ghost := adjacent interior value (slip).
 */
void wlo_bc(wlo_sim *s, double *u)
{
    const wlo_config *cf = &s->cfg;
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
    for (int j = 0; j < nd; ++j) {
        int N = g->n[j];
        long sj = g->st[j];
        int lo[3] = { 0, 0, 0 }, hi[3] = { g->S[0] - 1, g->S[1] - 1, g->S[2] - 1 };
        lo[j] = hi[j] = 0;
        for (int i = 0; i < nd; ++i) {
            double *a = u + i * nc;
            for (int c2 = lo[2]; c2 <= hi[2]; ++c2)
                for (int c1 = lo[1]; c1 <= hi[1]; ++c1)
                    for (int c0 = lo[0]; c0 <= hi[0]; ++c0) {
                        long b = IDX(g, c0, c1, c2);    /* c_j = 0 */
                        if (cf->periodic[j]) {
                            a[b] = a[b + N * sj];
                            a[b + (N + 1) * sj] = a[b + sj];
                        } else if (i == j) {
                            a[b] = cf->U[j];
                            a[b + sj] = cf->U[j];
                            if (!(cf->exit_bc && j == 0)) a[b + (N + 1) * sj] = cf->U[j];
                        } else {
                            a[b] = a[b + sj];
                            a[b + (N + 1) * sj] = a[b + N * sj];
                        }
                    }
        }
    }
}

/* -------------------------------------------------- O6: convective exit
 * P:139 "exitBC! ... implements a convective outlet".  Reading R-N: on the exit plane
 * c_x = N_x+1 (interior in the other directions)
 *   u_x <- u0_x[c] - U_x dt (u0_x[c] - u0_x[c-d_x]),
 * then subtract (mean_exit(u_x) - U_x) from every exit-plane value (global mass balance).
 */
void wlo_exit_bc(wlo_sim *s, double dt)
{
    const wlo_config *cf = &s->cfg;
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    int N = g->n[0];
    double sum = 0;
    long cnt = 0;
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1) {
            long id = IDX(g, N + 1, c1, c2);
            double v = s->u0[id] - cf->U[0] * dt * (s->u0[id] - s->u0[id - 1]);
            s->u[id] = v;
            sum += v;
            ++cnt;
        }
    double corr = sum / (double)cnt - cf->U[0];
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            s->u[IDX(g, N + 1, c1, c2)] -= corr;
}

/* -------------------------------------------------- O3: conv_diff
 * P:74 "Second-order central differences are used for the pressure and diffusion terms,
 * while a flux-limited Quick scheme is used on the convective term"; Eq. 1.
 * Reading R-G/H/I: flux through the LOWER j-boundary of the momentum control volume of
 * w_i[c] (valid for c_j = 1..N_j+1):
 *   phi = (w_j[c-d_i] + w_j[c])/2
 *   PHI = phi*psi - nu (w_i[c] - w_i[c-d_j])
 *   psi = q(w_i[c-2d_j], w_i[c-d_j], w_i[c])  if phi > 0 else q(w_i[c+d_j], w_i[c], w_i[c-d_j])
 *   q(U,C,D) = median((5C+2D-U)/6, C, median(10C-9U, C, D))
 * Non-periodic j: on c_j = 1 with phi > 0 and on c_j = N_j+1 with phi <= 0 the upwind
 * stencil would leave the padded array: psi = (w_i[c-d_j] + w_i[c])/2 there.  For the
 * normal component (i == j) the flux planes sit at cell centres, half a cell off the
 * tangential ones, and the plane c_j = 2 with phi > 0 is the mirror image of c_j = N_j+1
 * with phi <= 0; it takes the same 2-point value, so that the scheme commutes with a
 * reflection of the domain (reading R-H; pinned by test_sphere_flow_symmetry...).
 * Periodic directions: every index wraps into the interior.
 *   r_i[c] = sum_j PHI_j(c) - PHI_j(c+d_j)            (conservative: -d_j(u_j u_i) + nu d_jj u_i)
 * (SURVEY states the same sum in scatter form; the gather form used here evaluates the
 * same flux function on the same arguments for both cells sharing a boundary.)
 */
static inline double med3(double a, double b, double c)
{
    double lo = a < b ? a : b, hi = a < b ? b : a;
    return c < lo ? lo : (c > hi ? hi : c);
}
double wlo_quick(double U, double C, double D)
{
    return med3((5.0 * C + 2.0 * D - U) / 6.0, C, med3(10.0 * C - 9.0 * U, C, D));
}
static inline double WV(const wlo_sim *s, const double *w, int comp, int c0, int c1, int c2)
{
    const wlo_level *g = &s->lev[0];
    const int *per = s->cfg.periodic;
    c0 = wrapc(c0, g->n[0], per[0]);
    c1 = wrapc(c1, g->n[1], per[1]);
    if (s->nd == 3) c2 = wrapc(c2, g->n[2], per[2]);
    return w[comp * g->ncell + IDX(g, c0, c1, c2)];
}
static double cd_flux(const wlo_sim *s, const double *w, int i, int j, const int *c)
{
    int di[3] = { 0, 0, 0 }, dj[3] = { 0, 0, 0 };
    di[i] = 1; dj[j] = 1;
    int N = s->lev[0].n[j], per = s->cfg.periodic[j];
    double phi = 0.5 * (WV(s, w, j, c[0] - di[0], c[1] - di[1], c[2] - di[2]) + WV(s, w, j, c[0], c[1], c[2]));
    double wc = WV(s, w, i, c[0], c[1], c[2]);
    double wm = WV(s, w, i, c[0] - dj[0], c[1] - dj[1], c[2] - dj[2]);
    double psi;
    if (phi > 0) {
        if (!per && c[j] <= 1 + (i == j)) psi = 0.5 * (wm + wc);
        else psi = wlo_quick(WV(s, w, i, c[0] - 2 * dj[0], c[1] - 2 * dj[1], c[2] - 2 * dj[2]), wm, wc);
    } else {
        if (!per && c[j] == N + 1) psi = 0.5 * (wm + wc);
        else psi = wlo_quick(WV(s, w, i, c[0] + dj[0], c[1] + dj[1], c[2] + dj[2]), wc, wm);
    }
    return phi * psi - s->cfg.nu * (wc - wm);
}
void wlo_conv_diff(wlo_sim *s, const double *w, double *r)
{
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
    memset(r, 0, sizeof(double) * (size_t)nc * nd);
#pragma omp parallel for collapse(2) schedule(static)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                int c[3] = { c0, c1, c2 };
                for (int i = 0; i < nd; ++i) {
                    double acc = 0;
                    for (int j = 0; j < nd; ++j) {
                        int cp[3] = { c0, c1, c2 };
                        cp[j] += 1;
                        acc += cd_flux(s, w, i, j, c) - cd_flux(s, w, i, j, cp);
                    }
                    r[i * nc + id] = acc;
                }
            }
}

/* -------------------------------------------------- O4: BDIM blend
 * P:58-72, Eq. 1-2 "integrated in time and convolved with a prescribed body velocity ...
 * resulting in a single meta-equation".  Reading R-B/C (first-order expansion of the
 * eps-convolution in the normal direction):
 *   f = u0 + dt r - V   on the whole padded array (r = 0 in ghosts), ghosts of f wrapped
 *                       in periodic directions,
 *   B_i[c] = V_i + mu0[c,i] f_i[c] + sum_j mu1[c,i,j] (f_i[c+d_j] - f_i[c-d_j])/2 .
 * corr = 0: u = B (predictor);  corr = 1: u = (u + B)/2 (Heun average, O9 / scale_u! P:139).
 * On entry s->f holds r; on exit it holds f.
 */
void wlo_bdim(wlo_sim *s, double dt, int corr)
{
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
#pragma omp parallel for
    for (long k = 0; k < nc * nd; ++k) s->f[k] = s->u0[k] + dt * s->f[k] - s->V[k];
    for (int i = 0; i < nd; ++i) level_wrap(s, g, s->f + i * nc);
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                for (int i = 0; i < nd; ++i) {
                    const double *fi = s->f + i * nc;
                    double B = s->V[i * nc + id] + s->mu0[i * nc + id] * fi[id];
                    for (int j = 0; j < nd; ++j)
                        B += s->mu1[(i * nd + j) * nc + id] * 0.5 * (fi[id + g->st[j]] - fi[id - g->st[j]]);
                    s->u[i * nc + id] = corr ? 0.5 * (s->u[i * nc + id] + B) : B;
                }
            }
}

/* -------------------------------------------------- O7: Poisson operator
 * (A x)_c = sum_i L[c+d_i,i](x[c+d_i]-x[c]) - L[c,i](x[c]-x[c-d_i])   ("c are
 * the coefficients in the pressure-Poisson matrix").  Periodic ghosts of x are wrapped
 * before the mat-vec.  Returns sum_c q[c]*x[c] over the interior.
 */
static double level_matvec(const wlo_sim *s, const wlo_level *g, double *x, double *q)
{
    int nd = s->nd;
    double dot = 0;
    level_wrap(s, g, x);
#pragma omp parallel for collapse(2) reduction(+ : dot)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                double acc = 0;
                for (int i = 0; i < nd; ++i) {
                    const double *L = g->L + i * g->ncell;
                    long si = g->st[i];
                    acc += L[id + si] * (x[id + si] - x[id]) - L[id] * (x[id] - x[id - si]);
                }
                q[id] = acc;
                dot += acc * x[id];
            }
    return dot;
}

static double level_dot_riDr(const wlo_sim *s, const wlo_level *g, double *z)
{
    /* z = iD r ; returns r.z over the interior */
    int nd = s->nd;
    double dot = 0;
#pragma omp parallel for collapse(2) reduction(+ : dot)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                double zz = g->iD[id] * g->r[id];
                z[id] = zz;
                dot += zz * g->r[id];
            }
    return dot;
}

static double level_maxabs_r(const wlo_sim *s, const wlo_level *g)
{
    int nd = s->nd;
    double m = 0;
#pragma omp parallel for collapse(2) reduction(max : m)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                double a = fabs(g->r[IDX(g, c0, c1, c2)]);
                if (a > m) m = a;
            }
    return m;
}

/* -------------------------------------------------- O8: smoother
 * P:149 "a preconditioned conjugate gradient smoother (PCG) is employed in the geometric
 * multi-grid solver ... contains several reduction operations".  Reading R-S/T: Jacobi-
 * preconditioned CG, `its` iterations, restarted at every call:
 *   z = e = iD r; rho0 = rho = r.z; if |rho| < tau return
 *   loop k = 1..its: q = A e; gamma = q.e; (gamma = 0 or non-finite => return)
 *                    alpha = rho/gamma; x += alpha e; r -= alpha q; if k == its break;
 *                    z = iD r; rho' = r.z; if |rho'| < tau or |rho'| < theta |rho0| break;
 *                    beta = rho'/rho; e = beta e + z; rho = rho'
 * tau = 1e-30 only protects 0/0.  theta = 1e-8 stops the iteration once this call has reduced
 * the residual by 1e-4 in the iD norm: continuing CG on a converged residual divides round-off
 * by round-off (alpha = rho/gamma) and blows up -- in fp32 already on the 8x8 level of the
 * 2-D Taylor-Green case, whose residual is a single eigenmode (converged after two iterations).
 * A relative test makes the fp64 oracle and an fp32 implementation take the same branch.
 * Reading R-T2 (compatibility): A is singular -- constants span its null space, buried cells
 * (D = 0, iD = 0) are decoupled -- so A x = r has a solution only for a residual orthogonal to
 * the constants.  Before the iteration the mean of r over the coupled cells (iD != 0) is
 * removed from those cells.  In exact arithmetic that mean is zero (sum div u = boundary flux
 * = 0, sum A x = 0, restriction and prolongation preserve sums); in floating point it is
 * round-off, and CG on it diverges once the rest of r has converged below it (alpha = rho/gamma
 * with rho held up by the null-space part while gamma, which cannot see it, goes to zero).
 * `q` doubles as the z work array.
 */
#define WLO_TAU 1e-30
#define WLO_THETA 1e-8
void wlo_smooth(wlo_sim *s, int l, int its)
{
    wlo_level *g = &s->lev[l];
    int nd = s->nd;
    {   /* R-T2: r <- r - mean(r) over the coupled cells */
        double sum = 0, cnt = 0;
#pragma omp parallel for collapse(2) reduction(+ : sum, cnt)
        for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
            for (int c1 = 1; c1 <= g->n[1]; ++c1)
                for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                    long id = IDX(g, c0, c1, c2);
                    if (g->iD[id] != 0.0) { sum += g->r[id]; cnt += 1.0; }
                }
        double m = cnt > 0 ? sum / cnt : 0.0;
#pragma omp parallel for collapse(2)
        for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
            for (int c1 = 1; c1 <= g->n[1]; ++c1)
                for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                    long id = IDX(g, c0, c1, c2);
                    if (g->iD[id] != 0.0) g->r[id] -= m;
                }
    }
    double rho = level_dot_riDr(s, g, g->e);    /* z = e = iD r ; rho = r.z */
    double rho0 = rho;
    if (fabs(rho) < WLO_TAU) return;
    for (int k = 1; k <= its; ++k) {
        double gamma = level_matvec(s, g, g->e, g->q);  /* q = A e ; gamma = q.e */
        if (gamma == 0.0 || !isfinite(gamma)) return;
        double alpha = rho / gamma;
#pragma omp parallel for collapse(2)
        for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
            for (int c1 = 1; c1 <= g->n[1]; ++c1)
                for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                    long id = IDX(g, c0, c1, c2);
                    g->x[id] += alpha * g->e[id];
                    g->r[id] -= alpha * g->q[id];
                }
        if (k == its) break;
        double rho2 = level_dot_riDr(s, g, g->q);   /* z (in q) = iD r ; rho' = r.z */
        if (fabs(rho2) < WLO_TAU || fabs(rho2) < WLO_THETA * fabs(rho0)) break;
        double beta = rho2 / rho;
#pragma omp parallel for collapse(2)
        for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
            for (int c1 = 1; c1 <= g->n[1]; ++c1)
                for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                    long id = IDX(g, c0, c1, c2);
                    g->e[id] = beta * g->e[id] + g->q[id];
                }
        rho = rho2;
    }
}

/* residual restriction: r_c[C] = sum of the 2^n children (reading R-S) */
void wlo_restrict(wlo_sim *s, int l)
{
    const wlo_level *f = &s->lev[l];
    wlo_level *c = &s->lev[l + 1];
    int nd = s->nd;
#pragma omp parallel for collapse(2)
    for (int C2 = ZLO(c, nd); C2 <= ZHI(c, nd); ++C2)
        for (int C1 = 1; C1 <= c->n[1]; ++C1)
            for (int C0 = 1; C0 <= c->n[0]; ++C0) {
                double sum = 0;
                int n2 = nd == 3 ? 2 : 1;
                for (int a2 = 0; a2 < n2; ++a2)
                    for (int a1 = 0; a1 < 2; ++a1)
                        for (int a0 = 0; a0 < 2; ++a0)
                            sum += f->r[IDX(f, 2 * C0 - 1 + a0, 2 * C1 - 1 + a1, nd == 3 ? 2 * C2 - 1 + a2 : 0)];
                c->r[IDX(c, C0, C1, C2)] = sum;
            }
}

/* prolongation (piecewise constant): e_f[child] = x_c[parent]; then x_f += e_f,
 * r_f -= A_f e_f  (reading R-S) */
void wlo_prolong_increment(wlo_sim *s, int l)
{
    wlo_level *f = &s->lev[l];
    const wlo_level *c = &s->lev[l + 1];
    int nd = s->nd;
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(f, nd); c2 <= ZHI(f, nd); ++c2)
        for (int c1 = 1; c1 <= f->n[1]; ++c1)
            for (int c0 = 1; c0 <= f->n[0]; ++c0)
                f->e[IDX(f, c0, c1, c2)] = c->x[IDX(c, (c0 + 1) / 2, (c1 + 1) / 2, nd == 3 ? (c2 + 1) / 2 : 0)];
    level_matvec(s, f, f->e, f->q);
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(f, nd); c2 <= ZHI(f, nd); ++c2)
        for (int c1 = 1; c1 <= f->n[1]; ++c1)
            for (int c0 = 1; c0 <= f->n[0]; ++c0) {
                long id = IDX(f, c0, c1, c2);
                f->x[id] += f->e[id];
                f->r[id] -= f->q[id];
            }
}

/* V-cycle(l): restrict r_l -> r_{l+1}; x_{l+1} = 0; recurse unless l+1 is the coarsest;
 * smooth(l+1); prolong + increment.  No pre-smoothing (reading R-S). */
void wlo_vcycle(wlo_sim *s, int l)
{
    if (l + 1 >= s->nlev) return;
    wlo_level *c = &s->lev[l + 1];
    wlo_restrict(s, l);
    memset(c->x, 0, sizeof(double) * (size_t)c->ncell);
    if (l + 1 < s->nlev - 1) wlo_vcycle(s, l + 1);
    wlo_smooth(s, l + 1, s->cfg.smooth_iters);
    wlo_prolong_increment(s, l);
}

/* level-0 residual r = z - A x with z = s->sig */
void wlo_residual(wlo_sim *s)
{
    wlo_level *g = &s->lev[0];
    int nd = s->nd;
    level_matvec(s, g, g->x, g->q);
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                g->r[id] = s->sig[id] - g->q[id];
            }
}

/* solve A x = z on level 0 (reading R-S): r = z - A x; repeat { V-cycle(0); smooth(0) }
 * fixed_vcycles times, or until max|r| <= tol or max_vcycles. Returns V-cycles used. */
int wlo_solve(wlo_sim *s)
{
    const wlo_config *cf = &s->cfg;
    wlo_level *g = &s->lev[0];
    int nv = 0;
    wlo_residual(s);
    if (cf->fixed_vcycles > 0) {
        for (; nv < cf->fixed_vcycles; ++nv) {
            wlo_vcycle(s, 0);
            wlo_smooth(s, 0, cf->smooth_iters);
        }
    } else {
        while (level_maxabs_r(s, g) > cf->tol && nv < cf->max_vcycles) {
            wlo_vcycle(s, 0);
            wlo_smooth(s, 0, cf->smooth_iters);
            ++nv;
        }
    }
    s->last_res[s->solve_slot] = level_maxabs_r(s, g);
    s->last_vcycles[s->solve_slot] = nv;
    return nv;
}

/* -------------------------------------------------- O7: project(w)
 * P:76 "velocity is restricted to be incompressible using a pressure projection scheme";
 * P:88 the gradient update u[I,i] -= c[I,i]*(p[I]-p[I-d(i)]).
 *   z = div u, div_c = sum_i u_i[c+d_i] - u_i[c];  x = (w dt) p (warm start);
 *   solve A x = z;  u_i[c] -= L[c,i] (x[c] - x[c-d_i]);  p = x/(w dt).
 */
void wlo_divergence(wlo_sim *s, double *out)
{
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                double d = 0;
                for (int i = 0; i < nd; ++i) d += s->u[i * nc + id + g->st[i]] - s->u[i * nc + id];
                out[id] = d;
            }
}
void wlo_project(wlo_sim *s, double w, double dt)
{
    wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
    double sc = w * dt;
    wlo_divergence(s, s->sig);
#pragma omp parallel for
    for (long k = 0; k < nc; ++k) g->x[k] = sc * s->p[k];
    wlo_solve(s);
    level_wrap(s, g, g->x);
#pragma omp parallel for collapse(2)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                for (int i = 0; i < nd; ++i)
                    s->u[i * nc + id] -= g->L[i * nc + id] * (g->x[id] - g->x[id - g->st[i]]);
            }
#pragma omp parallel for
    for (long k = 0; k < nc; ++k) s->p[k] = g->x[k] / sc;
}

/* -------------------------------------------------- O9: mom_step (Heun)
 * P:76 "integrated in time using an explicit predictor-corrector update scheme"; routine
 * list P:139.  Reading R-K/L:
 *   u0 <- u
 *   predictor: r = conv_diff(u0); u = B(u0 + dt r); BC; exitBC; project(w=1); BC
 *   corrector: r = conv_diff(u);  u = (u + B(u0 + dt r))/2; BC; project(w=1/2); BC
 */
void wlo_mom_step(wlo_sim *s, double dt)
{
    const wlo_level *g = &s->lev[0];
    long nc = g->ncell;
    int nd = s->nd;
    memcpy(s->u0, s->u, sizeof(double) * (size_t)nc * nd);
    wlo_conv_diff(s, s->u0, s->f);
    wlo_bdim(s, dt, 0);
    wlo_bc(s, s->u);
    if (s->cfg.exit_bc) wlo_exit_bc(s, dt);
    s->solve_slot = 0;
    wlo_project(s, 1.0, dt);
    wlo_bc(s, s->u);
    wlo_conv_diff(s, s->u, s->f);
    wlo_bdim(s, dt, 1);
    wlo_bc(s, s->u);
    s->solve_slot = 1;
    wlo_project(s, 0.5, dt);
    wlo_bc(s, s->u);
}

/* -------------------------------------------------- O10: CFL
 * P:76 "time step is adapted automatically to ensure a stable CFL number".  Reading R-U:
 *   dt = min(dt_max, cfl_c / (max_c sum_i [max(0,u_i[c+d_i]) + max(0,-u_i[c])] + cfl_cnu nu))
 */
double wlo_cfl(wlo_sim *s)
{
    const wlo_level *g = &s->lev[0];
    const wlo_config *cf = &s->cfg;
    int nd = s->nd;
    long nc = g->ncell;
    double m = 0;
#pragma omp parallel for collapse(2) reduction(max : m)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                double a = 0;
                for (int i = 0; i < nd; ++i) {
                    double up = s->u[i * nc + id + g->st[i]], lo = s->u[i * nc + id];
                    a += (up > 0 ? up : 0) + (lo < 0 ? -lo : 0);
                }
                if (a > m) m = a;
            }
    double dt = cf->cfl_c / (m + cf->cfl_cnu * cf->nu);
    return dt < cf->dt_max ? dt : cf->dt_max;
}

/* -------------------------------------------------- O11: pressure force
 * P:175/P:181 use drag and power coefficients; the formula is not given.  Reading R-Z:
 *   F = - sum_{c interior} p[c] n(x_c) K^{eps_F}(d(x_c)),  eps_F = 1, at cell centres.
 */
void wlo_pressure_force(wlo_sim *s, double t, double *F)
{
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    double F0 = 0, F1 = 0, F2 = 0;
#pragma omp parallel for collapse(2) reduction(+ : F0, F1, F2)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                double xc[3] = { c0 - 0.5, c1 - 0.5, nd == 3 ? c2 - 0.5 : 0.0 }, nrm[3], vel[3];
                double d = wlo_body_eval(&s->cfg, xc, t, nrm, vel);
                double k = wlo_kernel_K(d, 1.0);
                if (k == 0.0) continue;
                double pk = s->p[IDX(g, c0, c1, c2)] * k;
                F0 -= pk * nrm[0]; F1 -= pk * nrm[1]; F2 -= pk * nrm[2];
            }
    F[0] = F0; F[1] = F1; F[2] = F2;
}

/* -------------------------------------------------- kinetic energy and enstrophy
 * P:169-173 (Fig. 4) follow the Taylor-Green vortex by its kinetic energy and enstrophy; the paper gives no
 * discrete formula.  Reading R-E2, the plain staggered-grid sums over the interior cells c (h = 1):
 *   KE = 1/2 sum_c sum_i u_i[c]^2                              (every face once: the lower faces of the cells)
 *   Z  = 1/2 sum_c |w[c]|^2,  w_k[c] = (u_j[c] - u_j[c - d_i]) - (u_i[c] - u_i[c - d_j]),  (i, j, k) cyclic,
 * the circulation around the cell edge along k through the lower-i, lower-j corner of cell c (2-D: w_z only).
 * Ghost values come from the BC fill.  out[0] = KE, out[1] = Z. */
void wlo_energy(wlo_sim *s, double *out)
{
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
    double ke = 0, ens = 0;
#pragma omp parallel for collapse(2) reduction(+ : ke, ens)
    for (int c2 = ZLO(g, nd); c2 <= ZHI(g, nd); ++c2)
        for (int c1 = 1; c1 <= g->n[1]; ++c1)
            for (int c0 = 1; c0 <= g->n[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                for (int i = 0; i < nd; ++i) ke += 0.5 * s->u[i * nc + id] * s->u[i * nc + id];
                for (int k = (nd == 3 ? 0 : 2); k < 3; ++k) {
                    int i = (k + 1) % 3, j = (k + 2) % 3;
                    double w = (s->u[j * nc + id] - s->u[j * nc + id - g->st[i]])
                             - (s->u[i * nc + id] - s->u[i * nc + id - g->st[j]]);
                    ens += 0.5 * w * w;
                }
            }
    out[0] = ke; out[1] = ens;
}

/* -------------------------------------------------- set-up */

/* TGV initial condition (Eq. 3-5 with the sign of BASELINE configs[0],[1];
 * reading R-W): u = s sin(kx)cos(ky)[cos(kz)], v = -s cos(kx)sin(ky)[cos(kz)], w = 0,
 * sampled at the staggered face positions; then BC fill.  k_d = 2 pi/N_d in a periodic direction (one
 * period in the box); k_d = pi/N_d in a non-periodic one: the box is then the half-period [0, pi] between
 * two symmetry planes of the vortex ("computational domain is the half-domain with symmetry boundary
 * conditions"), where the normal component vanishes and the tangential ones are even -- exactly what the
 * slip wall of reading R-M imposes when U = 0. */
void wlo_init_tgv(wlo_sim *s, int sign)
{
    const wlo_level *g = &s->lev[0];
    int nd = s->nd;
    long nc = g->ncell;
    const int *per = s->cfg.periodic;
    double k0 = (per[0] ? 2 : 1) * WLO_PI / g->n[0], k1 = (per[1] ? 2 : 1) * WLO_PI / g->n[1];
    double k2 = nd == 3 ? (per[2] ? 2 : 1) * WLO_PI / g->n[2] : 0;
    for (int c2 = 0; c2 < g->S[2]; ++c2)
        for (int c1 = 0; c1 < g->S[1]; ++c1)
            for (int c0 = 0; c0 < g->S[0]; ++c0) {
                long id = IDX(g, c0, c1, c2);
                double xc = c0 - 0.5, yc = c1 - 0.5, zc = nd == 3 ? c2 - 0.5 : 0.0;
                double cz = nd == 3 ? cos(k2 * zc) : 1.0;
                s->u[id] = sign * sin(k0 * (xc - 0.5)) * cos(k1 * yc) * cz;
                s->u[nc + id] = -sign * cos(k0 * xc) * sin(k1 * (yc - 0.5)) * cz;
                if (nd == 3) s->u[2 * nc + id] = 0.0;
            }
    memset(s->p, 0, sizeof(double) * (size_t)nc);
    wlo_bc(s, s->u);
}

static int config_ok(const wlo_config *cf)
{
    if (cf->ndim != 2 && cf->ndim != 3) return 0;
    for (int d = 0; d < cf->ndim; ++d) if (cf->dims[d] < 4) return 0;
    if (cf->nu < 0 || !(cf->eps > 0)) return 0;
    if (cf->body_kind < 0 || cf->body_kind > 4) return 0;
    if ((cf->body_kind == WLO_BODY_TORUS || cf->body_kind == WLO_BODY_CYLINDER) && (cf->ndim != 3 || cf->axis < 0 || cf->axis > 2)) return 0;
    if (cf->body_kind == WLO_BODY_PLANE && (cf->axis < 0 || cf->axis >= cf->ndim)) return 0;
    if (cf->nextra < 0 || cf->nextra > WLO_MAX_EXTRA || (cf->nextra > 0 && cf->body_kind == WLO_BODY_NONE)) return 0;
    for (int e = 0; e < cf->nextra; ++e) {
        const wlo_part *p = &cf->extra[e];
        if (p->kind < 1 || p->kind > 4 || p->axis < 0 || p->axis > 2) return 0;
        if ((p->kind == WLO_BODY_TORUS || p->kind == WLO_BODY_CYLINDER) && cf->ndim != 3) return 0;
    }
    return 1;
}

/* hierarchy rule (reading R-S): coarsen while every N_d is even and every N_d > 4,
 * capped by max_levels (<= 0 => uncapped). */
wlo_sim *wlo_create(const wlo_config *cf)
{
    if (!config_ok(cf)) return NULL;
    wlo_sim *s = (wlo_sim *)calloc(1, sizeof(wlo_sim));
    s->cfg = *cf;
    s->nd = cf->ndim;
    int nd = s->nd, n[3] = { cf->dims[0], cf->dims[1], nd == 3 ? cf->dims[2] : 1 };
    level_alloc(&s->lev[0], nd, n, 0);
    long nc = s->lev[0].ncell;
    s->u = (double *)calloc((size_t)nc * nd, sizeof(double));
    s->u0 = (double *)calloc((size_t)nc * nd, sizeof(double));
    s->f = (double *)calloc((size_t)nc * nd, sizeof(double));
    s->V = (double *)calloc((size_t)nc * nd, sizeof(double));
    s->mu0 = (double *)calloc((size_t)nc * nd, sizeof(double));
    s->mu1 = (double *)calloc((size_t)nc * nd * nd, sizeof(double));
    s->p = (double *)calloc((size_t)nc, sizeof(double));
    s->sig = (double *)calloc((size_t)nc, sizeof(double));
    s->lev[0].L = s->mu0;
    s->nlev = 1;
    int cap = cf->max_levels > 0 ? cf->max_levels : WLO_MAXLEV;
    if (cap > WLO_MAXLEV) cap = WLO_MAXLEV;
    while (s->nlev < cap) {
        int ok = 1;
        for (int d = 0; d < nd; ++d) if ((n[d] & 1) || n[d] <= 4) ok = 0;
        if (!ok) break;
        for (int d = 0; d < nd; ++d) n[d] /= 2;
        level_alloc(&s->lev[s->nlev], nd, n, 1);
        s->nlev++;
    }
    /* initial state (reading R-V): u = U everywhere, p = 0, measure(0) */
    for (int i = 0; i < nd; ++i)
        for (long k = 0; k < nc; ++k) s->u[i * nc + k] = cf->U[i];
    wlo_measure(s, 0.0);
    wlo_bc(s, s->u);
    return s;
}

void wlo_destroy(wlo_sim *s)
{
    if (!s) return;
    for (int l = 0; l < s->nlev; ++l) {
        wlo_level *g = &s->lev[l];
        if (l > 0) free(g->L);
        free(g->iD); free(g->x); free(g->r); free(g->e); free(g->q);
    }
    free(s->u); free(s->u0); free(s->f); free(s->V); free(s->mu0); free(s->mu1); free(s->p); free(s->sig);
    free(s);
}

/* ------------------------------------------------------------------ accessors for tests
 * name: "u","u0","f","p","sig","V","mu0","mu1" (level ignored) or level arrays
 * "L","iD","x","r","e","q".  shape[0] = number of components, shape[1..3] = S2,S1,S0. */
double *wlo_array(wlo_sim *s, const char *name, int level, int *shape)
{
    wlo_level *g = &s->lev[level];
    int nd = s->nd;
    double *p = NULL;
    int nc = 1;
    if (!strcmp(name, "u")) { p = s->u; nc = nd; g = &s->lev[0]; }
    else if (!strcmp(name, "u0")) { p = s->u0; nc = nd; g = &s->lev[0]; }
    else if (!strcmp(name, "f")) { p = s->f; nc = nd; g = &s->lev[0]; }
    else if (!strcmp(name, "V")) { p = s->V; nc = nd; g = &s->lev[0]; }
    else if (!strcmp(name, "mu0")) { p = s->mu0; nc = nd; g = &s->lev[0]; }
    else if (!strcmp(name, "mu1")) { p = s->mu1; nc = nd * nd; g = &s->lev[0]; }
    else if (!strcmp(name, "p")) { p = s->p; g = &s->lev[0]; }
    else if (!strcmp(name, "sig")) { p = s->sig; g = &s->lev[0]; }
    else if (!strcmp(name, "L")) { p = g->L; nc = nd; }
    else if (!strcmp(name, "iD")) p = g->iD;
    else if (!strcmp(name, "x")) p = g->x;
    else if (!strcmp(name, "r")) p = g->r;
    else if (!strcmp(name, "e")) p = g->e;
    else if (!strcmp(name, "q")) p = g->q;
    if (shape) { shape[0] = nc; shape[1] = g->S[2]; shape[2] = g->S[1]; shape[3] = g->S[0]; }
    return p;
}
int wlo_nlevels(const wlo_sim *s) { return s->nlev; }
void wlo_stats(const wlo_sim *s, int *vcycles, double *res)
{
    vcycles[0] = s->last_vcycles[0]; vcycles[1] = s->last_vcycles[1];
    res[0] = s->last_res[0]; res[1] = s->last_res[1];
}
/* level mat-vec exposed for the operator pins: q = A_level x, returns q.x */
double wlo_matvec(wlo_sim *s, int level, double *x, double *q)
{
    return level_matvec(s, &s->lev[level], x, q);
}
void wlo_poisson_update(wlo_sim *s) { poisson_update(s); }
int wlo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
