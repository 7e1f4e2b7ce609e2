"""Seeded synthetic inputs and the workload catalogue, shared by the oracle tests, the GPU
parity tests and bench.py.

This module holds NONE of the method's arithmetic (no stencils, kernels, SDFs, solvers):
only plain parameter dictionaries (the five BASELINE.json configs in grid units, see
DESIGN.md section 4) and a seeded random-field generator.  Both the oracle binding
(oracle/wl_oracle.py) and the CUDA binding (paper_2407_16032_b200/wl.py) turn these
dictionaries into their own config structs.
"""
from __future__ import annotations

import math

import numpy as np

SEED = 20240716  # per-kernel parity inputs

BODY_NONE, BODY_SPHERE, BODY_TORUS, BODY_CYLINDER, BODY_PLANE = 0, 1, 2, 3, 4
MOTION_STATIC, MOTION_SIN = 0, 1
MOTION_HEAVE_SIN = MOTION_SIN          # one direction of the sinusoidal translation (heave_dir, amp, freq, phase)

CONFIG_DEFAULTS = dict(
    ndim=3, dims=(32, 32, 32), L=1.0, U=(1.0, 0.0, 0.0), nu=0.01,
    periodic=(0, 0, 0), exit_bc=0, eps=1.0,
    dt0=0.25, dt_max=10.0, cfl_c=1.0, cfl_cnu=5.0,
    body_kind=BODY_NONE, centre=(0.0, 0.0, 0.0), R=0.0, r=0.0, axis=0,
    motion=MOTION_STATIC, heave_dir=1, amp=0.0, freq=0.0, phase=0.0,
    amp3=None, freq3=None, phase3=None,     # sinusoidal translation in every direction (overrides the four above)
    tune=None,                              # implementation switches of the CUDA library (wl_tuning), a dict
    # general bodies: thin shell |sdf| - shell, non-rigid map xi_d = s_d(t)(x_d - c_d(t)) with
    # s_d = 1 + scale_amp[d] cos(2 pi scale_freq t + scale_phase), spin about the axis, and further primitives combined by
    # SDF arithmetic: parts = [dict(kind=..., centre=..., ..., op="+" | "-"), ...] (same keys as the first primitive)
    shell=0.0, scale_amp=(0.0, 0.0, 0.0), scale_freq=0.0, scale_phase=0.0, spin=0.0, parts=None,
    # scalar type of the CUDA library: precision 1 = fp64; tangent = (parameter name, index): the
    # forward-mode derivative of the whole step with respect to "nu" | "U" | "R" | "spin" | "amp" | "centre"
    precision=0, tangent=None,
    max_levels=0, smooth_iters=6, max_vcycles=32, fixed_vcycles=2, tol=1e-4,
)


def make(**kw) -> dict:
    cfg = dict(CONFIG_DEFAULTS)
    for k, v in kw.items():
        if k not in cfg:
            raise KeyError(k)
        cfg[k] = v
    return cfg


def tgv2d(n=64, nu_phys=0.01, **kw) -> dict:
    """C1: 2-D Taylor-Green vortex on [0,2pi)^2, n x n periodic; grid units h = 2pi/n."""
    h = 2 * math.pi / n
    base = dict(ndim=2, dims=(n, n), L=n / (2 * math.pi), U=(0.0, 0.0, 0.0), nu=nu_phys / h,
                periodic=(1, 1), max_levels=4)
    base.update(kw)
    return make(**base)


def tgv3d(n=128, Re=1600.0, **kw) -> dict:
    """C2: 3-D Taylor-Green vortex, n^3 periodic, Re = U L_ref / nu with L_ref = 1/kappa."""
    Lref = n / (2 * math.pi)
    base = dict(ndim=3, dims=(n, n, n), L=Lref, U=(0.0, 0.0, 0.0), nu=Lref / Re, periodic=(1, 1, 1))
    base.update(kw)
    return make(**base)


def sphere(dims=(256, 128, 128), D=32.0, Re=3700.0, centre=None, **kw) -> dict:
    """C3: static sphere, inflow +x, convective exit, slip side walls."""
    centre = centre or (dims[0] / 4.0, dims[1] / 2.0, dims[2] / 2.0)
    base = dict(ndim=3, dims=tuple(dims), L=D, U=(1.0, 0.0, 0.0), nu=D / Re, exit_bc=1,
                body_kind=BODY_SPHERE, centre=tuple(centre), R=D / 2.0)
    base.update(kw)
    return make(**base)


def torus(dims=(512, 256, 256), R=32.0, r=8.0, Re=1000.0, centre=None, **kw) -> dict:
    """C4: static torus, axis along the inflow, Re on the minor diameter 2r."""
    centre = centre or (dims[0] / 4.0, dims[1] / 2.0, dims[2] / 2.0)
    base = dict(ndim=3, dims=tuple(dims), L=2 * r, U=(1.0, 0.0, 0.0), nu=2 * r / Re, exit_bc=1,
                body_kind=BODY_TORUS, centre=tuple(centre), R=R, r=r, axis=0)
    base.update(kw)
    return make(**base)


def heaving_sphere(dims=(384, 256, 256), D=48.0, Re=1000.0, St=0.2, amp_over_D=0.25, centre=None, **kw) -> dict:
    """C5: sphere heaving in y, y(t) = amp sin(2 pi f t), St = f D / U."""
    centre = centre or (dims[0] / 3.0, dims[1] / 2.0, dims[2] / 2.0)
    base = dict(ndim=3, dims=tuple(dims), L=D, U=(1.0, 0.0, 0.0), nu=D / Re, exit_bc=1,
                body_kind=BODY_SPHERE, centre=tuple(centre), R=D / 2.0,
                motion=MOTION_HEAVE_SIN, heave_dir=1, amp=amp_over_D * D, freq=St / D)
    base.update(kw)
    return make(**base)


def cylinder_2dof(L=64, Re=1000.0, **kw) -> dict:
    """SURVEY 8(f) NEXT-1, the paper's third benchmark case: circular cylinder of diameter L cells
    spanning the periodic z direction of a 9L x 6L x 2L box, inflow +x, convective exit, slip in y, Re = U L / nu,
    with the prescribed two-degree-of-freedom motion of PAPER.md:181: y = A_y sin(w t), x = A_x sin(2 w t + theta),
    A_y = 1.6 D, A_x = 0.4 D, theta = pi/6, w = (2 pi / 5.4) U / D.  The paper does not say where the cylinder
    sits in the benchmark box: centre (3L, 3L) here."""
    D = float(L)
    f = 1.0 / (5.4 * D)
    base = dict(ndim=3, dims=(9 * L, 6 * L, 2 * L), L=D, U=(1.0, 0.0, 0.0), nu=D / Re, periodic=(0, 0, 1), exit_bc=1,
                body_kind=BODY_CYLINDER, axis=2, centre=(3.0 * L, 3.0 * L, 0.0), R=D / 2.0, motion=MOTION_SIN,
                amp3=(0.4 * D, 1.6 * D, 0.0), freq3=(2.0 * f, f, 0.0), phase3=(math.pi / 6.0, 0.0, 0.0))
    base.update(kw)
    return make(**base)


def jelly(p=5, Re=500.0, U=1.0, **kw) -> dict:
    """SURVEY 8(f) NEXT-2, the pulsing jellyfish of PAPER.md:235-243: a spherical shell |  |xi| - R | - 1 under the non-rigid map
    xi = A(t) .* x + B(t) + C(t), minus the half-space xi_3 < h under the translation x + C(t) ("body = sphere - plane"), in a
    box n x n x 4n with n = 2^p, R = 2n/3, h = 4n - 2R, nu = U R / Re, omega = 2U/R, boundary velocity (0, 0, -U):
        A = 1 - [1,1,0] 0.1 cos(wt),  B = [0,0,1] ((cos(wt) - 1) R/4 - h),  C = [0,0,1] sin(wt) R/4.
    In this module's parametrisation xi_d = s_d(t)(x_d - c_d(t)): s = A, c = -(B + C) ./ A, i.e. for the sphere
    c_z = h + R/4 - (R sqrt(2)/4) sin(wt + pi/4); for the plane c_z = -C_z... (xi_3 - h = x_3 + C_z - h): c_z = h - (R/4) sin(wt)."""
    n = 2 ** p
    R = 2.0 * n / 3.0
    h = 4.0 * n - 2.0 * R
    w = 2.0 * U / R
    f = w / (2.0 * math.pi)
    base = dict(ndim=3, dims=(n, n, 4 * n), L=R, U=(0.0, 0.0, -U), nu=U * R / Re, periodic=(0, 0, 0), exit_bc=0,
                body_kind=BODY_SPHERE, centre=(0.0, 0.0, h + R / 4.0), R=R, shell=1.0, motion=MOTION_SIN,
                amp3=(0.0, 0.0, -R * math.sqrt(2.0) / 4.0), freq3=(0.0, 0.0, f), phase3=(0.0, 0.0, math.pi / 4.0),
                scale_amp=(-0.1, -0.1, 0.0), scale_freq=f, scale_phase=0.0,
                parts=[dict(kind=BODY_PLANE, axis=2, centre=(0.0, 0.0, h), motion=MOTION_SIN,
                            amp3=(0.0, 0.0, -R / 4.0), freq3=(0.0, 0.0, f), phase3=(0.0, 0.0, 0.0), op="-")])
    base.update(kw)
    return make(**base)


def control_cylinders(D=32, Re=500.0, xi=3.0, **kw) -> dict:
    """SURVEY 8(f) NEXT-2, the controlled cylinder of PAPER.md:202-210 ("body = big + small"): a circle of diameter D with a small
    spinning circle (d/D = 0.15, gap g/D = 0.05, surface speed xi U = d Omega / 2) placed 120 degrees from the inflow
    direction, upper half of the flow only (symmetry plane y = 0), 2-D box 6D x 2D."""
    d, gap = 0.15 * D, 0.05 * D
    rc = D / 2.0 + gap + d / 2.0
    ang = math.radians(120.0)                         # measured from the upstream direction (-x)
    cx, cy = 2.0 * D, 0.0
    sx, sy = cx - rc * math.cos(ang), cy + rc * math.sin(ang)
    base = dict(ndim=2, dims=(6 * D, 2 * D), L=float(D), U=(1.0, 0.0), nu=D / Re, periodic=(0, 0), exit_bc=1,
                body_kind=BODY_SPHERE, centre=(cx, cy), R=D / 2.0,
                parts=[dict(kind=BODY_SPHERE, centre=(sx, sy), R=d / 2.0, spin=-2.0 * xi / d, op="+")])
    base.update(kw)
    return make(**base)


def tgv3d_half(n=512, Re=1600.0, **kw) -> dict:
    """SURVEY 8(f) NEXT-3, the paper's first benchmark case as it states it: the Taylor-Green vortex on
    the half-domain [0, pi]^3 of n^3 cells between symmetry planes (slip walls with U = 0), kappa = pi / n,
    Re = U / (kappa nu)."""
    Lref = n / math.pi
    base = dict(ndim=3, dims=(n, n, n), L=Lref, U=(0.0, 0.0, 0.0), nu=Lref / Re, periodic=(0, 0, 0))
    base.update(kw)
    return make(**base)


def baseline_config(k: int, scale: int = 1) -> dict:
    """BASELINE.json configs[k]; scale > 1 divides every length by `scale` (same shape,
    same Reynolds number) for tests the oracle must finish in seconds."""
    s = scale
    if k == 0:
        return tgv2d(64 // s)
    if k == 1:
        return tgv3d(128 // s)
    if k == 2:
        return sphere((256 // s, 128 // s, 128 // s), D=32.0 / s, centre=(64.0 / s, 64.0 / s, 64.0 / s))
    if k == 3:
        return torus((512 // s, 256 // s, 256 // s), R=32.0 / s, r=8.0 / s,
                     centre=(128.0 / s, 128.0 / s, 128.0 / s))
    if k == 4:
        return heaving_sphere((384 // s, 256 // s, 256 // s), D=48.0 / s,
                              centre=(128.0 / s, 128.0 / s, 128.0 / s))
    raise IndexError(k)


WORKLOAD_NAMES = ["C1_tgv2d_64", "C2_tgv3d_128", "C3_sphere_256x128x128",
                  "C4_torus_512x256x256", "C5_heaving_sphere_384x256x256"]


def rng(seed: int = SEED) -> np.random.Generator:
    return np.random.Generator(np.random.MT19937(seed))


def random_velocity(dims, seed: int = SEED, nmodes: int = 8, kmax: int = 4, step: float = 0.5,
                    mean=(1.0, 0.0, 0.0)) -> np.ndarray:
    """Interior-sized velocity (ndim, [Nz,] Ny, Nx), float64: a sum of `nmodes` random
    Fourier modes (|k| <= kmax, amplitudes U(-0.5,0.5)) + a uniform stream + a planar step
    of height `step` at x = N/3 (exercises both limiter branches and both flux signs)."""
    g = rng(seed)
    nd = len(dims)
    shape = tuple(reversed(dims))
    axes = [np.arange(n, dtype=np.float64) for n in dims]           # x, y[, z]
    grids = np.meshgrid(*reversed(axes), indexing="ij")               # z, y, x order
    grids = list(reversed(grids))                                     # -> x, y[, z]
    u = np.zeros((nd,) + shape)
    for c in range(nd):
        for _ in range(nmodes):
            k = g.integers(-kmax, kmax + 1, size=nd)
            amp = g.uniform(-0.5, 0.5)
            ph = g.uniform(0, 2 * math.pi)
            arg = ph
            for d in range(nd):
                arg = arg + 2 * math.pi * k[d] * grids[d] / dims[d]
            u[c] += amp * np.sin(arg)
        u[c] += mean[c] if c < len(mean) else 0.0
    u[0] += step * (grids[0] >= dims[0] / 3.0)
    return u


def random_scalar(dims, seed: int = SEED + 1, nmodes: int = 8, kmax: int = 4) -> np.ndarray:
    """Interior-sized scalar ([Nz,] Ny, Nx), float64, random Fourier modes + white noise."""
    g = rng(seed)
    nd = len(dims)
    shape = tuple(reversed(dims))
    axes = [np.arange(n, dtype=np.float64) for n in dims]
    grids = list(reversed(np.meshgrid(*reversed(axes), indexing="ij")))
    a = np.zeros(shape)
    for _ in range(nmodes):
        k = g.integers(-kmax, kmax + 1, size=nd)
        amp = g.uniform(-0.5, 0.5)
        ph = g.uniform(0, 2 * math.pi)
        arg = ph
        for d in range(nd):
            arg = arg + 2 * math.pi * k[d] * grids[d] / dims[d]
        a += amp * np.sin(arg)
    a += 0.1 * g.standard_normal(shape)
    return a
