/*
 * wl.h -- C ABI of libwl: one incompressible BDIM time step (mom_step) on a B200.
 *
 * The operations are the routines the paper names for one time step of its solver
 * (/root/reference/PAPER.md, cited "P:<line>"; Fig. 2 caption P:139 lists them:
 * measure!, conv_diff!, BDIM!, BC!, exitBC!, scale_u!, project!, CFL!), on the uniform
 * staggered Cartesian grid of P:74 with the boundary-data-immersion treatment of P:58-72
 * (Eq. 1-2).  The paper defers every formula to cited works; the readings this library
 * implements are written out in DESIGN.md section 3 ("R-<x>") and restate SURVEY.md 8(c).
 *
 * Conventions
 *   - plain C, no exceptions, no global state; every call returns an int status
 *     (WL_OK = 0, negative = error) unless stated otherwise.
 *   - one handle = one CUDA stream; calls on one handle are not thread-safe.
 *   - DEVICE memory is owned by the caller: the workspace passed to wl_sim_create is
 *     allocated by the caller (through PyTorch in this repo), must be 256-byte aligned,
 *     must outlive the handle, and is never freed by the library.
 *   - grid units: spacing h = 1, density 1 ("no grid information is stored");
 *     cell c (1-based interior index I_d = 2..N_d+1 in the paper) has centre
 *     x = I_d - 3/2; u_i[I] lives on the LOWER i-face of cell I (forced by the stencil of
 *     the pressure-gradient kernel u[I,i] -= c[I,i]*(p[I]-p[I-d(i)])).
 *   - user-visible field buffers are INTERIOR-sized, x fastest: a scalar is
 *     dims[2]*dims[1]*dims[0] floats (2-D: dims[1]*dims[0]); a vector field is ndim such
 *     arrays back to back (component-major).  `on_device` says whether the pointer is a
 *     device (1) or host (0) pointer.
 *   - all arithmetic is fp32 on the device; reductions accumulate in fp64.
 *   - there is no CPU fallback: every entry point that computes runs CUDA kernels.
 */
#ifndef WL_H
#define WL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* status codes */
#define WL_OK        0
#define WL_EINVAL   -1   /* bad argument / config (ndim not 2 or 3, a dim < 4, nu < 0, eps <= 0, unknown body) */
#define WL_ENOMEM   -2   /* workspace too small or misaligned */
#define WL_ECUDA    -3   /* CUDA error (sticky); text through wl_last_error */
#define WL_ENOCONV  -4   /* tolerance-mode Poisson solve hit max_vcycles (result still written) */
#define WL_ETOOBIG  -5   /* wl_energy_static: the grid exceeds WL_STATIC_MAX_CELLS */

/* body kinds and motions: SDF + coordinate map of the paper's AutoBody.
 * WL_BODY_CYLINDER is the circular cylinder of P:121 / P:179 (radius R, infinitely long along `axis`: it spans a
 * periodic direction).  WL_MOTION_SIN is a rigid translation, sinusoidal in every direction:
 *     c_d(t) = centre[d] + amp[d] sin(2 pi freq[d] t + phase[d]),   V_d = dc_d/dt  (uniform in space),
 * which covers the heaving sphere (one non-zero amp) and the two-degree-of-freedom cylinder of P:181,
 * y = A_y sin(w t), x = A_x sin(2 w t + theta). */
enum { WL_BODY_NONE = 0, WL_BODY_SPHERE = 1 /* circle in 2-D */, WL_BODY_TORUS = 2, WL_BODY_CYLINDER = 3,
       WL_BODY_PLANE = 4 /* half-space below the plane through `centre` with normal +e_axis */ };
enum { WL_MOTION_STATIC = 0, WL_MOTION_SIN = 1 };
enum { WL_OP_UNION = 0, WL_OP_DIFFERENCE = 1 };
#define WL_MAX_EXTRA 3

/* One primitive: SDF + map.  General bodies (reading R-E3 of DESIGN.md):
 *   map       xi_d = s_d(t) (x_d - c_d(t)),  s_d(t) = 1 + scale_amp[d] cos(2 pi scale_freq t + scale_phase)   ("A(t) .* x + B(t)");
 *   shell > 0 the body is the thin shell |sdf| - shell around the primitive's surface;
 *   normal    J^T grad sdf / |J^T grad sdf|, distance sdf / |J^T grad sdf| when the map is non-rigid, J = diag(s);
 *   velocity  V = -J^-1 dmap/dt = dc/dt - (ds/dt / s) .* (x - c), plus spin e_axis x (x - c) (z axis in 2-D): a body of
 *             revolution spinning about its axis keeps its SDF, not its surface velocity. */
typedef struct {
    int   kind;          /* WL_BODY_* */
    float centre[3];     /* c0, grid units */
    float R, r;          /* sphere / cylinder radius R; torus major R, minor r */
    int   axis;          /* torus / cylinder / plane axis 0..2 */
    int   motion;        /* WL_MOTION_* */
    float amp[3], freq[3], phase[3];
    float shell;
    float scale_amp[3], scale_freq, scale_phase;
    float spin;
} wl_body;

typedef struct {
    int   max_levels;    /* <= 0: coarsen while every N_d is even and > 4 */
    int   smooth_iters;  /* Jacobi-PCG iterations per smoother call */
    int   max_vcycles;   /* tolerance mode cap */
    int   fixed_vcycles; /* > 0: exactly this many {V-cycle; smooth} per solve, no tolerance test */
    float tol;           /* tolerance mode: stop when max|r| <= tol */
} wl_mg;

/* Implementation switches, for A/B tests of alternative kernel paths (tests/test_gpu_paths.py) and tuning runs.
 * All zero = the defaults.  Part of the config so that a handle carries no hidden state: the library reads no
 * environment variable. */
typedef struct {
    int no_fused;        /* PCG smoother as two passes per iteration instead of the one-sweep form (wl_pcgfused.cu) */
    int no_fast_a;       /* register-marching pass A everywhere (no shared-memory kernel) */
    int no_bulk;         /* pass A stages its planes with per-thread cp.async instead of TMA boxes */
    int no_block_levels; /* small levels by the cooperative kernel instead of the one-block kernel */
    int no_tma_cd;       /* conv_diff from the register-staged ring (k_cd_tile2) instead of the TMA-fed one */
    int zc;              /* planes per tile of the vector kernels (0: 8) */
    long long pk_max_cells; /* levels >= 1 with at most this many cells run inside the persistent kernels (0: 2^20; < 0: none) */
    int pk_blocks_per_sm;   /* co-resident blocks per SM of the cooperative kernel (0: 2) */
    int pk_fail;            /* test hook: treat the first cooperative / cluster launch as refused by the device (exercises the fallback) */
} wl_tuning;

/* Problem statement (grid size, boundary velocity, length scale, viscosity, BC type,
 * body).  POD, caller-owned, copied at create. */
typedef struct {
    int   ndim;          /* 2 or 3 */
    int   dims[3];       /* interior cells N_d (dims[2] ignored in 2-D) */
    float L;             /* length scale; only scales reported quantities */
    float U[3];          /* boundary / inflow velocity */
    float nu;            /* kinematic viscosity in grid units */
    int   periodic[3];   /* per direction; a non-periodic direction is a slip wall with normal velocity U_d: with
                            U_d = 0 that is the symmetry plane of P:118 (normal component 0, tangential mirrored) */
    int   exit_bc;       /* convective exit on the +x plane */
    float eps;           /* BDIM kernel half-width in cells */
    float dt0, dt_max, cfl_c, cfl_cnu;   /* CFL rule, DESIGN.md R-U */
    wl_body body;
    wl_mg   mg;
    wl_tuning tune;
    /* SDF arithmetic ("body = big + small", "body = sphere - plane"): the body is
     * ((body op[0] extra[0]) op[1] extra[1]) ..., union = min of the distances, difference = max(d, -d_extra); normal and
     * velocity are those of the primitive that decides.  With more than one primitive, a non-rigid map or spin the body
     * velocity is a per-face field (one more array of ndim components); otherwise three scalars. */
    int     nextra;
    wl_body extra[WL_MAX_EXTRA];
    int     extra_op[WL_MAX_EXTRA];   /* WL_OP_* */
    /* Scalar type of the simulation ("T=Float32"; "T = Dual"):
     *   precision = 0        fp32, the tuned kernels (the hot path this library is about);
     *   precision = 1        fp64, through the generic engine (one plain kernel per stage, same algorithm);
     *   tangent_param != 0   forward-mode tangent: every kernel of the step carries d/d(theta) beside the value (fp64 dual
     *                        numbers, generic engine), theta = the parameter named by WL_SEED_* (tangent_index: the direction
     *                        for U / AMP / CENTRE, the primitive 0..nextra for SPIN).  dt is taken as independent of theta.
     * The generic engine supports every entry point except the wl_dbg_* stage hooks and wl_prof_*; wl_step's device-resident
     * dt becomes a host round trip per step. */
    int     precision;
    int     tangent_param;
    int     tangent_index;
} wl_config;

enum { WL_SEED_NONE = 0, WL_SEED_NU = 1, WL_SEED_U = 2, WL_SEED_R = 3, WL_SEED_SPIN = 4, WL_SEED_AMP = 5, WL_SEED_CENTRE = 6 };

typedef struct wl_sim wl_sim;

typedef struct {
    int    vcycles[2];   /* V-cycles used by the predictor / corrector solve of the last step */
    double res[2];       /* max|r| after each (tolerance mode only; -1 in fixed mode) */
    int    nlevels;
    int    kernel_launches;   /* kernels launched by this handle since create */
    int    nan_flag;          /* 1 if the last CFL reduction saw a non-finite velocity */
    int    noconv;            /* tolerance-mode solves since create that hit max_vcycles (WL_ENOCONV is also
                                 returned, once, by the next wl_cfl) */
} wl_stats_t;

/* Pure function: bytes of device workspace wl_sim_create needs; 0 on invalid config. */
size_t wl_workspace_bytes(const wl_config* cfg);

/* Create a simulation in caller-owned DEVICE memory `dev_ws` (>= wl_workspace_bytes,
 * 256-B aligned).  `cuda_stream` is a cudaStream_t (NULL = default stream).  Initial state
 * (R-V): u = U everywhere, p = 0, measure(0), multigrid hierarchy built, BC filled. */
int wl_sim_create(const wl_config* cfg, void* dev_ws, size_t ws_bytes, void* cuda_stream, wl_sim** out);

/* Frees the host-side handle only (never the workspace).  Synchronises the stream. */
int wl_sim_destroy(wl_sim* s);

/* Set state from interior-sized buffers (NULL leaves a field untouched); u: ndim arrays,
 * p: one.  Ghost cells are then filled by the BC rule.  Synchronises when host. */
int wl_set_fields(wl_sim* s, const float* u, const float* p, int on_device);

/* Taylor-Green initial condition of P:112-116 (Eq. 3-5), staggered sampling; sign = +1 gives BASELINE.json's
 * u = sin x cos y [cos z], v = -cos x sin y [cos z]; sign = -1 gives the paper's.  One period of the vortex in every
 * periodic direction, half a period in every non-periodic one (the half-domain between symmetry planes of P:118:
 * use U = 0).  p = 0. */
int wl_init_tgv(wl_sim* s, int sign);

/* measure!: evaluate the SDF and motion map at every face at time t (solver
 * time units h/U), write mu0, mu1, body velocity V, then the Poisson diagonal and the
 * coarse-level coefficients.  Call before wl_mom_step when the body moves (R-R:
 * with t = t_n + dt).  Asynchronous. */
int wl_measure(wl_sim* s, double t);

/* mom_step ("explicit predictor-corrector", routine list P:139; reading R-K):
 * one full Heun step with two pressure projections.  Asynchronous on the stream. */
int wl_mom_step(wl_sim* s, float dt);

/* CFL! ("time step is adapted automatically"): dt for the next step from the current
 * velocity (reading R-U).  Synchronises. */
int wl_cfl(wl_sim* s, float* dt_out);

/* Pressure force ON THE BODY, grid units (rho = 1, h = 1), reading R-Z:
 * F = -sum_cells p n K(d) at cell centres, body placed at time t (NaN: where the last measure! placed it).  Neither
 * the stored body state nor the simulation time changes.  Synchronises. */
int wl_pressure_force(wl_sim* s, double t, float F_out[3]);

/* Kinetic energy and enstrophy of the current velocity (Fig. 4 follows the Taylor-Green vortex by them;
 * reading R-E2): out[0] = 1/2 sum_cells sum_i u_i^2, out[1] = 1/2 sum_cells |w|^2 with w the circulations around the
 * cell edges through the lower corner of each cell, grid units.  fp64 partial sums, fixed tree.  Synchronises. */
int wl_energy(wl_sim* s, double out[2]);

/* Copy interior fields out; any pointer may be NULL.  u: ndim arrays; p, mu0 likewise
 * (mu0: ndim arrays).  Synchronises when host. */
int wl_get_fields(wl_sim* s, float* u, float* p, float* mu0, int on_device);

/* fp64 views of the state for the fp64 and tangent modes (generic engine only: WL_EINVAL otherwise).  tangent = 0: the
 * values; 1: the derivatives d/d(theta) (tangent mode only).  Interior-sized buffers as wl_get_fields. */
int wl_get_fields_f64(wl_sim* s, double* u, double* p, int tangent, int on_device);
int wl_set_fields_f64(wl_sim* s, const double* u, const double* p, int on_device);
/* pressure force and its derivative (dF may be NULL; zero in fp64 mode) */
int wl_pressure_force_f64(wl_sim* s, double t, double F[3], double dF[3]);
/* kinetic energy, enstrophy and their derivatives (dout may be NULL) */
int wl_energy_f64(wl_sim* s, double out[2], double dout[2]);
/* interior copy of a solver array ("u","p","mu0","mu1","V","L","iD","x","r") as doubles into a HOST buffer; returns ncomp */
int wl_dbg_get_f64(wl_sim* s, const char* name, int level, int tangent, double* out, size_t out_doubles);

/* Fused step: wl_measure(t) (only if the body moves) + wl_mom_step(dt) + the CFL reduction, all asynchronous; t is
 * the time the step ends at (R-R) and becomes the simulation time.  With `adaptive` != 0 the NEXT call ignores `t` and
 * `dt` and uses the device-resident CFL result and simulation time + dt (no host round trip). */
int wl_step(wl_sim* s, double t, float dt, int adaptive);

/* ---- stage hooks: each applies one stage once to the current state (parity tests) ---- */
int wl_dbg_conv_diff_bdim(wl_sim* s, float dt, int corrector); /* u0 must hold the step's start state: see wl_dbg_save_u0 */
int wl_dbg_save_u0(wl_sim* s);                                 /* u0 <- u */
int wl_dbg_bc(wl_sim* s);
int wl_dbg_exit_bc(wl_sim* s, float dt);
int wl_dbg_project(wl_sim* s, float w, float dt);
int wl_dbg_residual(wl_sim* s);                                /* sigma = div u; r = sigma - A x on level 0 */
int wl_dbg_apply_gradient(wl_sim* s);                          /* P:88 kernel with the current x and pscale: u -= L grad x; p = x/pscale */
int wl_dbg_restrict(wl_sim* s, int level);
int wl_dbg_prolong(wl_sim* s, int level);
int wl_dbg_smooth(wl_sim* s, int level, int iters);
int wl_dbg_vcycle(wl_sim* s, int level);
/* Runs n coarse-level passes as one chain through the persistent kernels: kinds[k] = 0 restrict
 * levels[k] -> levels[k]+1, 1 smooth level levels[k] with iters[k] PCG iterations, 2 prolong levels[k]+1 -> levels[k].
 * Consecutive passes of the same kind of launch share a launch.  n <= 48. */
int wl_dbg_coarse_prog(wl_sim* s, int n, const int* kinds, const int* levels, const int* iters);
/* Device-resident PCG scalars of a level: rho, gamma, alpha, beta, rho0, sum of r over the coupled cells (R-T2),
 * number of coupled cells, live flag.  Synchronises. */
int wl_dbg_pcg_scalars(wl_sim* s, int level, double out[8]);
/* Raw access to a solver array for tests: name in {"u","u0","p","mu0","mu1","V" (general bodies only),"L","iD","x","r"};
 * interior-sized copy into `out` (host), ncomp arrays; returns ncomp or a negative status. */
int wl_dbg_get(wl_sim* s, const char* name, int level, float* out, size_t out_floats);
int wl_dbg_set(wl_sim* s, const char* name, int level, const float* in, size_t in_floats);
/* same as wl_dbg_get but the whole padded array (ghost cells included): (N_d + 2) per direction */
int wl_dbg_get_padded(wl_sim* s, const char* name, int level, float* out, size_t out_floats);
int wl_level_dims(const wl_sim* s, int level, int dims_out[3]);

/* Per-kernel-class timing for bench.py's roofline figure.  With enable != 0
 * every kernel the handle launches is bracketed by two CUDA events on its stream; enabling or
 * disabling synchronises and discards earlier records.  wl_prof_read synchronises and returns,
 * for class `cls` = 0, 1, ..., the class name (kernel name; ".coarse" = multigrid levels > 0),
 * the summed device time in ms and the number of launches since wl_prof_enable.  Returns 1
 * (not an error) once `cls` is past the last class. */
int wl_prof_enable(wl_sim* s, int enable);
int wl_prof_read(wl_sim* s, int cls, char* name_out, size_t name_bytes, double* ms_total, int* launches);

/* ---- the one entry point that ALLOCATES NOTHING (wl_noalloc.cu), for callers that cannot call cudaMalloc: code under
 * CUDA-graph capture, tight serving loops, harnesses that forbid it.  No handle, no workspace.
 * Kinetic energy and enstrophy as wl_energy defines them (reading R-E2) of a velocity field the CALLER holds:
 *   u_dev   device; ndim component arrays (u_x, u_y[, u_z]) of (dims[0]+2)(dims[1]+2)[(dims[2]+2)] floats each, x fastest, WITH
 *           the one-cell ghost layer around the interior filled by the caller (the paper's array layout; what
 *           wl_dbg_get_padded returns); read only, stays the caller's;
 *   dims    host; interior cells per direction, each >= 1; their product may not exceed WL_STATIC_MAX_CELLS;
 *   out_dev device; two doubles written: out[0] = 1/2 sum_cells sum_i u_i^2, out[1] = 1/2 sum_cells |w|^2 (fp32 products,
 *           fp64 sums in a fixed order);
 *   err     host, may be NULL; receives a text when the call fails (err_len bytes at most).
 * Asynchronous on `cuda_stream` (one memset node + one kernel: capturable); does not synchronise.  Returns WL_OK, WL_EINVAL
 * (bad argument), WL_ETOOBIG (more than WL_STATIC_MAX_CELLS cells: nothing is launched) or WL_ECUDA.
 * The reduction scratch (a pair of partial sums per 1024 cells + a ticket counter) is a file-scope __device__ array of
 * 1 MiB + 256 B that every GPU which loads libwl holds until the process exits.  ALL calls on a device share it: calls that
 * overlap on the GPU (different streams or host threads) race on it and return garbage; calls on one stream are safe.  It
 * keeps the last call's contents; the call clears what must start at zero.  The first call on a device looks the array's
 * address up (cudaGetSymbolAddress): make that call outside a stream capture. */
#define WL_STATIC_MAX_CELLS (64ll * 1024 * 1024)
int wl_energy_static(const float* u_dev, int ndim, const int* dims, void* cuda_stream, double* out_dev, char* err, size_t err_len);

const char* wl_last_error(const wl_sim* s);
int wl_stats(wl_sim* s, wl_stats_t* out);
int wl_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WL_H */
