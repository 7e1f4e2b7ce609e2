"""GPU parity of the generic engine (wl_generic.cu; SURVEY 8(f) NEXT-5 fp64 mode, NEXT-4 forward-mode tangent).

fp64 mode: the same step in double precision against the fp64 oracle -- the two differ by summation order only, so they
agree to ~1e-12 per step where the tuned fp32 kernels agree to ~1e-6.

Tangent mode: every kernel carries d/d(theta) beside the value ("the exact derivative, not a finite-
difference approximation").  The value lane must equal the fp64 mode's; the derivative lane is compared with a central
finite difference of the ORACLE in theta (the oracle has no derivative code: two runs at theta +- h), for theta = nu, the
inflow speed, the body radius, the heave amplitude and the spin rate of the control circle."""
import numpy as np
import pytest

import wl_inputs as wi

pytestmark = pytest.mark.gpu


def _f32(v):
    """wl_config stores its parameters as C floats: give the oracle the same (rounded) numbers, or the two solve problems that
    differ by 1e-7 -- invisible to the fp32 kernels, six orders above the agreement of the fp64 mode"""
    if isinstance(v, float):
        return float(np.float32(v))
    if isinstance(v, (tuple, list)):
        return type(v)(_f32(x) for x in v)
    if isinstance(v, dict):
        return {k: _f32(x) for k, x in v.items()}
    return v


def O(o, name):
    a = o.interior(name)
    return a[:, 0] if o.nd == 2 else a


def _run_oracle(cfg, steps, dt, tgv=False, force_t=None):
    from oracle import wl_oracle as wo
    o = wo.OracleSim(cfg)
    if tgv:
        o.init_tgv(1)
    moving = cfg["motion"] != wi.MOTION_STATIC or cfg.get("parts")
    t = 0.0
    for _ in range(steps):
        if moving:
            o.measure(t + dt)
        o.mom_step(dt)
        t += dt
    out = (O(o, "u").copy(), O(o, "p")[0].copy(), o.pressure_force(t) if cfg["body_kind"] else np.zeros(3), o.energy())
    o.close()
    return out


def _run_gpu(cfg, steps, dt, tgv=False):
    from paper_2407_16032_b200 import wl
    g = wl.Sim(cfg)
    if tgv:
        g.init_tgv(1)
    moving = cfg["motion"] != wi.MOTION_STATIC or cfg.get("parts")
    t = 0.0
    for _ in range(steps):
        if moving:
            g.measure(t + dt)
        g.mom_step(dt)
        t += dt
    return g, t


FP64_CASES = {
    "C1_tgv2d_64": (lambda: wi.baseline_config(0), True),
    "C3_sphere_64x32x32": (lambda: wi.baseline_config(2, scale=4), False),
    "C5_heaving_48x32x32": (lambda: wi.baseline_config(4, scale=8), False),
    "N1_cylinder_2dof_72x48x16": (lambda: wi.cylinder_2dof(8), False),
    "N2_jelly_16x16x64": (lambda: wi.jelly(4), False),
    "2d_control_cylinders_96x32": (lambda: wi.control_cylinders(16), False),
}


@pytest.mark.parametrize("name", list(FP64_CASES))
def test_fp64_mode_matches_the_oracle(name):
    mk, tgv = FP64_CASES[name]
    cfg = dict(_f32(mk()), precision=1)
    dt = cfg["nu"] if name.startswith("C1") else 0.25
    uo, po, Fo, eo = _run_oracle(cfg, 5, dt, tgv)
    g, t = _run_gpu(cfg, 5, dt, tgv)
    u, p = g.fields_f64()
    assert np.abs(u - uo).max() <= 1e-9 * np.abs(uo).max()
    F, _ = g.pressure_force_f64(t)
    assert np.abs(F - Fo).max() <= 1e-8 * max(np.abs(Fo).max(), 1e-30)
    e, _ = g.energy_f64()
    assert np.allclose(e, eo, rtol=1e-8)
    assert g.cfl() > 0 and g.stats()["vcycles"] == [2, 2] and g.stats()["nan_flag"] == 0
    # the float32 views of the same state
    uf, pf = g.fields()
    assert np.abs(uf - u).max() <= 1e-6 * np.abs(u).max()
    g.close()


def _f32_except(cfg, seed, theta):
    """every parameter rounded to float EXCEPT the one the derivative is taken with respect to (theta +- h must survive);
    theta itself is chosen exactly representable"""
    out = _f32(cfg)
    name, idx = seed
    if name == "nu":
        out["nu"] = theta
    elif name == "U":
        out["U"] = tuple(theta if k == idx else v for k, v in enumerate(out["U"]))
    elif name == "R":
        out["R"] = theta
    elif name == "amp":
        out["amp"] = theta
    elif name == "spin":
        out["parts"][idx - 1]["spin"] = theta
    return out


def _fd(cfg_of, theta, h, steps, dt, tgv=False):
    a = _run_oracle(cfg_of(theta + h), steps, dt, tgv)
    b = _run_oracle(cfg_of(theta - h), steps, dt, tgv)
    return [(x - y) / (2 * h) for x, y in zip(a, b)]


def _with_part(cfg, **kw):
    parts = [dict(cfg["parts"][0], **kw)] + list(cfg["parts"][1:])
    return dict(cfg, parts=parts)


TANGENT_CASES = {
    # name: (config as a function of theta, theta, h, seed)
    "nu_tgv2d_32": (lambda th: wi.tgv2d(32, nu_phys=0.01, nu=th), 0.046875, 1e-6, ("nu", 0), True),
    "nu_sphere_48x24x24": (lambda th: wi.sphere((48, 24, 24), D=8.0, centre=(12.0, 12.0, 12.0), nu=th), 0.01953125, 1e-6, ("nu", 0), False),
    "U_sphere_48x24x24": (lambda th: wi.sphere((48, 24, 24), D=8.0, centre=(12.0, 12.0, 12.0), nu=0.02, U=(th, 0.0, 0.0)), 1.0, 1e-6, ("U", 0), False),
    "R_circle_64x32": (lambda th: wi.make(ndim=2, dims=(64, 32), exit_bc=1, nu=0.05, body_kind=wi.BODY_SPHERE, centre=(20.3, 16.2), R=th), 5.0, 1e-6, ("R", 0), False),
    "amp_heaving_48x32x32": (lambda th: dict(wi.baseline_config(4, scale=8), amp=th), 1.5, 1e-6, ("amp", 1), False),
    # derivative of the flow (and of the force) with respect to the spin rate of the control circle
    "spin_control_cylinders_96x32": (lambda th: _with_part(wi.control_cylinders(16), spin=th), -2.5, 1e-6, ("spin", 1), False),
}


@pytest.mark.parametrize("name", list(TANGENT_CASES))
def test_tangent_matches_finite_differences_of_the_oracle(name):
    cfg_of, theta, h, seed, tgv = TANGENT_CASES[name]
    steps, dt = 4, 0.25
    cfg_raw = cfg_of
    cfg_of = lambda th: _f32_except(cfg_raw(th), seed, th)
    cfg = dict(cfg_of(theta), tangent=seed)
    uo, po, Fo, eo = _run_oracle(cfg_of(theta), steps, dt, tgv)
    du_fd, dp_fd, dF_fd, de_fd = _fd(cfg_of, theta, h, steps, dt, tgv)
    g, t = _run_gpu(cfg, steps, dt, tgv)
    u, p = g.fields_f64()
    du, dp = g.fields_f64(tangent=True)
    assert np.abs(u - uo).max() <= 1e-9 * np.abs(uo).max()                 # the value lane is the fp64 step
    scale = np.abs(du_fd).max()
    assert scale > 1e-6                                                    # the parameter does act on the flow
    # central differences with h = 1e-6 in fp64: truncation ~h^2, round-off ~1e-16/h -> 1e-9 absolute on O(1) data; a flux-
    # limiter branch that flips between theta - h and theta + h shows up as an isolated outlier: the 99.99th percentile
    err = np.abs(du - du_fd)
    assert np.percentile(err, 99.99) <= 1e-5 * scale, (np.percentile(err, 99.99), scale)
    assert np.median(err) <= 1e-7 * scale
    F, dF = g.pressure_force_f64(t)
    if cfg["body_kind"]:
        assert np.abs(F - Fo).max() <= 1e-8 * np.abs(Fo).max()
        assert np.abs(dF - dF_fd).max() <= 1e-4 * max(np.abs(dF_fd).max(), 1e-12)
    e, de = g.energy_f64()
    assert np.allclose(de, de_fd, rtol=1e-4, atol=1e-6 * abs(eo[0]))
    g.close()


def test_generic_engine_refuses_the_stage_hooks_and_reports_its_modes():
    from paper_2407_16032_b200 import wl
    g = wl.Sim(dict(wi.baseline_config(2, scale=8), precision=1))
    with pytest.raises(wl.WLError):
        g.dbg_residual()
    with pytest.raises(wl.WLError):
        g.fields_f64(tangent=True)                  # no derivative lane in plain fp64 mode
    g.step(0.25, 0.25, adaptive=True)
    g.step(0.0, 0.25, adaptive=True)                # the CFL result of the first step, through the host
    assert g.stats()["kernel_launches"] > 0
    g.close()
    f = wl.Sim(wi.baseline_config(2, scale=8))
    with pytest.raises(wl.WLError):
        f.fields_f64()                              # the tuned fp32 path has no fp64 view
    f.close()
