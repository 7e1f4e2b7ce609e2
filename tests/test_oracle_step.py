"""Pins for the oracle's O9 (mom_step), O10 (CFL), O11 (pressure force): the closed-form
decay of the 2-D Taylor-Green vortex, its pressure field, second-order convergence in
space and time, exact free-stream preservation, symmetry invariants with a body, CFL
closed forms and the divergence-theorem value of the force integral.  CPU only."""
import math

import numpy as np
import pytest

import wl_inputs as wi
from golden_util import load
from oracle import wl_oracle as wo

G = load()


def _run_tgv2d(n, steps, dt, **kw):
    cfg = wi.tgv2d(n, fixed_vcycles=0, tol=1e-10, max_vcycles=100, **kw)
    s = wo.OracleSim(cfg)
    s.init_tgv(1)
    u0 = s.interior("u").copy()
    for _ in range(steps):
        s.mom_step(dt)
    return s, u0, cfg


def test_ghost_layout_matches_paper():
    """size(p) == (10,10) -> inside(p) = 2:9 (1-based) == C indices 1..8."""
    s = wo.OracleSim(wi.make(ndim=2, dims=(8, 8), periodic=(1, 1)))
    assert s.arr("p").shape[1:] == (1, 10, 10)
    assert s.interior("p").shape[2:] == (8, 8)
    lo, hi = int(G["inside_size10_lo"]), int(G["inside_size10_hi"])
    assert (lo - 1, hi - 1) == (1, 8)
    s.close()


def test_tgv_initial_field_is_discretely_divergence_free():
    for cfg in (wi.tgv2d(64), wi.tgv3d(16), wi.make(ndim=3, dims=(16, 16, 12), periodic=(1, 1, 1))):   # needs N_x == N_y
        s = wo.OracleSim(cfg)
        s.init_tgv(1)
        assert np.abs(s.divergence()).max() < 5e-15
        s.init_tgv(-1)                              # the paper's sign (Eq. 3-5) as well
        assert np.abs(s.divergence()).max() < 5e-15
        s.close()


def test_tgv2d_closed_form_decay_C1():
    """BASELINE configs[0] / north_star pin: 64x64, nu = 0.01, dt = 0.01 (physical), 20 steps:
    amplitude = exp(-2 nu k^2 t) = exp(-0.004)."""
    cfg0 = wi.tgv2d(64)
    dt = cfg0["nu"]                                  # 0.01 / h  (nu_phys = dt_phys = 0.01)
    assert dt == pytest.approx(0.1018592, rel=1e-6)
    s, u0, cfg = _run_tgv2d(64, 20, dt)
    u = s.interior("u")
    amp = (u * u0).sum() / (u0 * u0).sum()
    assert amp == pytest.approx(G["tgv2d_c1_decay_20"], rel=1e-4)
    # the field keeps its shape: u = amp * u0 pointwise
    assert np.abs(u - amp * u0).max() < 5e-4       # limiter clips at the extrema
    assert np.abs(s.divergence()).max() < 1e-9
    s.close()


def test_tgv2d_pressure_closed_form():
    """p -> (cos 2kx + cos 2ky)/4 * amp^2 up to a constant (sign and the w*dt scaling of p)."""
    n = 64
    s, u0, cfg = _run_tgv2d(n, 3, 0.1)
    k = 2 * math.pi / n
    c = np.arange(n) + 0.5
    X, Y = np.meshgrid(c, c, indexing="xy")
    amp2 = math.exp(-2 * cfg["nu"] * k * k * 0.3) ** 2
    pex = 0.25 * (np.cos(2 * k * X) + np.cos(2 * k * Y)) * amp2
    p = s.interior("p")[0, 0]
    p = p - p.mean()
    assert np.abs(p - pex).max() < 0.02 * np.abs(pex).max()
    s.close()


def test_tgv2d_second_order_in_space():
    """Error in the decay factor falls ~4x per refinement at fixed physical time and dt ~ h."""
    errs = []
    for n in (16, 32, 64):
        h = 2 * math.pi / n
        nu = 0.05 / h
        dt = 0.05 / h * (16 / n)                    # physical dt = 0.05 * 16/n
        steps = 4 * n // 16                          # physical t = 0.2
        s, u0, cfg = _run_tgv2d(n, steps, dt, nu=nu)
        u = s.interior("u")
        amp = (u * u0).sum() / (u0 * u0).sum()
        errs.append(abs(amp - math.exp(-2 * 0.05 * 0.2)))
        s.close()
    assert errs[0] / errs[1] > 3.0 and errs[1] / errs[2] > 3.0


def test_heun_second_order_in_time():
    """Richardson on a smooth scalar functional (projection of u on the initial field) at a fixed
    final time: (a_dt - a_dt/2) / (a_dt/2 - a_dt/4) ~ 4 (spatial error cancels).  A pointwise max
    norm is too noisy here because the limiter's medians make the flux only Lipschitz."""
    n, T = 32, 2.4
    cfg = wi.tgv2d(n, fixed_vcycles=0, tol=1e-12, max_vcycles=200, nu=0.2)
    amps = []
    for steps in (8, 16, 32):
        s = wo.OracleSim(cfg)
        s.set_fields(u=wi.random_velocity((n, n), seed=17, mean=(0.3, 0.1), step=0.0, kmax=2))
        s.project(1.0, 1.0)
        s.bc()
        s.arr("p")[...] = 0
        u0 = s.interior("u").copy()
        for _ in range(steps):
            s.mom_step(T / steps)
        amps.append((s.interior("u") * u0).sum() / (u0 * u0).sum())
        s.close()
    ratio = (amps[0] - amps[1]) / (amps[1] - amps[2])
    assert 3.2 < ratio < 4.8


@pytest.mark.parametrize("n,nudt", [(8, 0.1), (8, 0.2), (16, 0.2)])
def test_heun_stability_polynomial(n, nudt):
    """Closed form: a low-amplitude 2-D TGV is an eigenfunction of the 5-point Laplacian with
    eigenvalue -lam = -2(2 - 2cos k), convection is O(amplitude^2), so one Heun step multiplies it
    by exactly 1 - z + z^2/2 with z = nu dt lam (explicit Euler would give 1 - z, the exact flow
    exp(-z)).  Fixes the two-stage structure and the 1/2 average of O9."""
    k = 2 * math.pi / n
    z = nudt * 2 * (2 - 2 * math.cos(k))
    dt = 0.5
    cfg = wi.tgv2d(n, fixed_vcycles=0, tol=1e-13, max_vcycles=200)
    cfg["nu"] = nudt / dt
    s = wo.OracleSim(cfg)
    s.init_tgv(1)
    s.arr("u")[...] *= 1e-4
    u0 = s.interior("u").copy()
    for _ in range(5):
        s.mom_step(dt)
    u = s.interior("u")
    amp = (u * u0).sum() / (u0 * u0).sum()
    heun, euler, exact = (1 - z + z * z / 2) ** 5, (1 - z) ** 5, math.exp(-5 * z)
    assert abs(amp - heun) < 2e-5
    assert abs(amp - euler) > 1e-3 and abs(amp - exact) > 1e-4 or n == 16
    assert np.abs(u - amp * u0).max() < 1e-5 * np.abs(u0).max()
    s.close()


@pytest.mark.parametrize("nd", [2, 3])
def test_uniform_free_stream_preserved_exactly(nd):
    """BASELINE north_star pin: no body, inflow / convective exit / slip walls: u stays exactly
    U and p stays exactly 0."""
    dims = (24, 16) if nd == 2 else (24, 12, 8)
    cfg = wi.make(ndim=nd, dims=dims, periodic=(0,) * 3, exit_bc=1, U=(1.0, 0.0, 0.0), nu=0.01)
    s = wo.OracleSim(cfg)
    dt = cfg["dt0"]
    for _ in range(5):
        s.mom_step(dt)
        dt = s.cfl()
    u = s.arr("u")
    assert np.all(u[0] == 1.0) and np.all(u[1:] == 0.0) and np.all(s.arr("p") == 0.0)
    assert dt == pytest.approx(1.0 / (1.0 + 5 * 0.01))
    s.close()


def test_sphere_flow_symmetry_and_force_components():
    """C3-shaped case (scaled 1/8): the grid, body and BCs are mirror-symmetric in y and z
    about the body centre, so the fields are too and F_y = F_z = 0 to round-off."""
    cfg = wi.baseline_config(2, scale=8)            # 32 x 16 x 16, D = 4
    s = wo.OracleSim(cfg)
    dt = cfg["dt0"]
    t = 0.0
    for _ in range(10):
        s.mom_step(dt)
        t += dt
        dt = s.cfl()
    u = s.interior("u")
    assert np.abs(u[0] - u[0][:, ::-1, :]).max() < 1e-11
    assert np.abs(u[0] - u[0][::-1, :, :]).max() < 1e-11
    p = s.interior("p")[0]
    assert np.abs(p - p[:, ::-1, :]).max() < 1e-10
    F = s.pressure_force(t)
    assert abs(F[1]) < 1e-10 and abs(F[2]) < 1e-10
    assert F[0] > 0.0                                # drag pushes the body downstream
    # no-slip / no-penetration: velocity deep inside the body is V = 0
    # (R = 2: the only faces deeper than eps = 1 inside are the ones through the centre cell corner)
    assert np.abs(u[:, 8, 8, 8]).max() < 1e-12
    assert np.abs(s.divergence()[0, 1:-1, 1:-1, 1:-1]).max() < 0.05
    s.close()


def test_impulsive_start_added_mass():
    """Weak physical check (SURVEY 8(c) pins, O9+body): in the first step of an impulsively started
    flow the pressure sets up the potential flow round the sphere, whose impulse is the added mass
    times U: F_x dt = (1/2)(4/3 pi R^3) U (textbook added-mass coefficient of a sphere; the far field
    never accelerates, so there is no buoyancy-like term).  Within 10% at D = 16; also fixes the sign
    and the 1/(w dt) scaling of p."""
    cfg = wi.sphere((64, 48, 48), D=16.0, centre=(24.0, 24.0, 24.0), fixed_vcycles=0, tol=1e-6, max_vcycles=60)
    s = wo.OracleSim(cfg)
    dt = 0.25
    s.mom_step(dt)
    F = s.pressure_force(dt)
    vol = 4.0 / 3.0 * math.pi * 8.0 ** 3
    assert F[0] * dt == pytest.approx(0.5 * vol, rel=0.10)
    s.close()


# ------------------------------------------------------------------ O10
def test_cfl_closed_forms():
    cfg = wi.make(ndim=3, dims=(8, 8, 8), periodic=(1, 1, 1), U=(0.0,) * 3, nu=0.0)
    s = wo.OracleSim(cfg)
    s.arr("u")[0][...] = 2.0
    s.arr("u")[1:][...] = 0.0
    assert s.cfl() == pytest.approx(1.0 / 2.0)      # uniform (U,0,0), nu = 0: dt = cfl_c / U
    s.arr("u")[0][...] = 4.0
    assert s.cfl() == pytest.approx(1.0 / 4.0)      # u -> 2u halves dt
    s.arr("u")[...] = 0.0
    assert s.cfl() == 10.0                          # dt_max cap
    s.close()
    cfg = wi.make(ndim=2, dims=(8, 8), periodic=(1, 1), U=(0.0,) * 3, nu=0.3)
    s = wo.OracleSim(cfg)
    s.arr("u")[...] = 0.0
    assert s.cfl() == pytest.approx(1.0 / (5 * 0.3))
    # outflow from one cell through both x faces and the upper y face: sum of outgoing fluxes
    u = s.arr("u")
    u[0][0, 4, 4] = -0.5     # lower x face, pointing out
    u[0][0, 4, 5] = 0.7      # upper x face, pointing out
    u[1][0, 5, 4] = 0.2      # upper y face, pointing out
    u[1][0, 4, 4] = 0.9      # lower y face, pointing IN: not counted for this cell
    # cell (4,4): 0.5+0.7+0.2 = 1.4 ; cell (3,4) sees 0.9 out through its upper y face only
    assert s.cfl() == pytest.approx(1.0 / (1.4 + 1.5))
    s.close()


# ------------------------------------------------------------------ O11
def test_pressure_force_divergence_theorem():
    """p = const => F ~ 0;  p = g x => F = -g Vol e_x (sign and magnitude; O(h^2) error)."""
    R = 16.0
    cfg = wi.sphere((48, 48, 48), D=2 * R, centre=(24.0, 24.0, 24.0))
    s = wo.OracleSim(cfg)
    vol = 4.0 / 3.0 * math.pi * R ** 3
    s.arr("p")[...] = 3.0
    F = s.pressure_force(0.0)
    assert np.abs(F).max() < 1e-9 * vol
    xc = np.arange(50) - 0.5
    s.arr("p")[0][...] = 0.01 * xc[None, None, :]
    F = s.pressure_force(0.0)
    assert F[0] == pytest.approx(-0.01 * vol, rel=0.01)
    assert abs(F[1]) < 1e-9 * vol and abs(F[2]) < 1e-9 * vol
    s.arr("p")[0][...] = -0.02 * xc[None, :, None]
    F = s.pressure_force(0.0)
    assert F[1] == pytest.approx(0.02 * vol, rel=0.01)
    s.close()


def test_pressure_force_moving_body_uses_time():
    cfg = wi.heaving_sphere((32, 32, 32), D=12.0, centre=(16.0, 16.0, 16.0), amp_over_D=0.25, St=0.3)
    s = wo.OracleSim(cfg)
    yc = np.arange(34) - 0.5
    s.arr("p")[0][...] = 0.01 * yc[None, :, None]
    vol = 4.0 / 3.0 * math.pi * 6.0 ** 3
    for t in (0.0, 10.0, 30.0):
        F = s.pressure_force(t)
        assert F[1] == pytest.approx(-0.01 * vol, rel=0.03)
    s.close()
