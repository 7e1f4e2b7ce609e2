"""Pins for the oracle's general bodies (reading R-E3): thin shells, the non-rigid diagonal map
xi = s(t) .* (x - c(t)) of PAPER.md:235-239, spin, the half-space primitive and SDF arithmetic ("body = big +
small", "body = sphere - plane").  Closed forms, finite differences of the map itself, and the paper's own listing of
the jellyfish evaluated directly in numpy.  CPU only."""
import math

import numpy as np
import pytest

import wl_inputs as wi
from oracle import wl_oracle as wo


def test_uniformly_scaled_sphere_is_a_sphere_of_radius_R_over_s():
    """s_x = s_y = s_z = s(t): the body is the sphere |x - c| = R/s exactly, so d = |x - c| - R/s (the first-order distance
    d0/|grad d0| is exact here), n radial, V = dc/dt - (ds/dt / s)(x - c)."""
    cfg = wi.make(ndim=3, dims=(32, 32, 32), body_kind=wi.BODY_SPHERE, centre=(15.0, 16.0, 17.0), R=6.0, motion=wi.MOTION_SIN,
                  amp3=(1.0, 2.0, 0.0), freq3=(0.02, 0.01, 0.0), phase3=(0.3, 0.0, 0.0),
                  scale_amp=(0.2, 0.2, 0.2), scale_freq=0.03, scale_phase=0.4)
    g = wi.rng(3)
    for t in (0.0, 4.2, 17.0):
        s = 1 + 0.2 * math.cos(2 * math.pi * 0.03 * t + 0.4)
        sd = -0.2 * 2 * math.pi * 0.03 * math.sin(2 * math.pi * 0.03 * t + 0.4)
        c = np.array([15 + math.sin(2 * math.pi * 0.02 * t + 0.3), 16 + 2 * math.sin(2 * math.pi * 0.01 * t), 17.0])
        cd = np.array([2 * math.pi * 0.02 * math.cos(2 * math.pi * 0.02 * t + 0.3), 2 * 2 * math.pi * 0.01 * math.cos(2 * math.pi * 0.01 * t), 0.0])
        for _ in range(10):
            x = c + g.uniform(-12, 12, 3)
            d, n, v = wo.body_eval(cfg, x, t)
            rr = np.linalg.norm(x - c)
            assert d == pytest.approx(rr - 6.0 / s, abs=1e-12)
            assert np.allclose(n, (x - c) / rr, atol=1e-12)
            assert np.allclose(v, cd - (sd / s) * (x - c), atol=1e-12)


def _material_point_velocity(cfg, x, t, h=1e-5):
    """d/dt of the position of the material point that sits at x at time t, from the MAP alone: xi = s(t) (x - c(t)) is fixed,
    so x(t') = c(t') + xi / s(t').  c and s are read back from the config (the parametrisation of wl_inputs.make)."""
    def cs(tt):
        c = np.array(cfg["centre"], dtype=float)
        amp, freq, ph = (cfg["amp3"], cfg["freq3"], cfg["phase3"]) if cfg["amp3"] is not None else wo.wi_motion(cfg)
        c = c + np.array(amp) * np.sin(2 * math.pi * np.array(freq) * tt + np.array(ph))
        s = 1 + np.array(cfg["scale_amp"]) * math.cos(2 * math.pi * cfg["scale_freq"] * tt + cfg["scale_phase"])
        return c, s
    c0, s0 = cs(t)
    xi = s0 * (np.array(x) - c0)
    xp = [cc + xi / ss for cc, ss in (cs(t + h), cs(t - h))]
    return (xp[0] - xp[1]) / (2 * h)


def test_nonrigid_map_normal_distance_and_velocity_by_finite_differences():
    """The jellyfish bell without its plane: n = grad_x d0 / |grad_x d0| and d = d0 / |grad_x d0| with
    d0(x) = | |s .* (x - c)| - R | - 1 differentiated numerically; V against the motion of a material point."""
    cfg = wi.jelly(4, parts=None)
    R = cfg["R"]

    def d0(x, t):
        c = np.array(cfg["centre"]) + np.array(cfg["amp3"]) * np.sin(2 * math.pi * np.array(cfg["freq3"]) * t + np.array(cfg["phase3"]))
        s = 1 + np.array(cfg["scale_amp"]) * math.cos(2 * math.pi * cfg["scale_freq"] * t + cfg["scale_phase"])
        return abs(np.linalg.norm(s * (np.array(x) - c)) - R) - 1.0

    g = wi.rng(8)
    for t in (0.0, 3.1, 9.9):
        for _ in range(20):
            x = np.array([g.uniform(0, 16), g.uniform(0, 16), g.uniform(30, 64)])
            d, n, v = wo.body_eval(cfg, x, t)
            h = 1e-6
            grad = np.array([(d0(x + h * e, t) - d0(x - h * e, t)) / (2 * h) for e in np.eye(3)])
            m = np.linalg.norm(grad)
            assert np.allclose(n, grad / m, atol=1e-6) and np.linalg.norm(n) == pytest.approx(1.0, abs=1e-12)
            assert d == pytest.approx(d0(x, t) / m, abs=1e-6)
            assert np.allclose(v, _material_point_velocity(cfg, x, t), atol=1e-7)


def test_jelly_parametrisation_is_the_papers_listing():
    """wl_inputs.jelly against the listing of PAPER.md:235-243 evaluated directly: sphere sdf abs(sqrt(sum(abs2, xi))) - R) - 1 at
    xi = A .* x + B + C, plane sdf xi_3 - h at xi = x + C, body = sphere - plane = max(d_sphere, -d_plane).  Compared at times
    where cos(w t) = 0, when A = 1 and the map is a pure translation (so that the normalised distance IS the listing's sdf)."""
    p = 4
    cfg = wi.jelly(p)
    n = 2 ** p
    R = 2 * n / 3
    h = 4 * n - 2 * R
    w = 2 * 1.0 / R
    assert cfg["dims"] == (n, n, 4 * n) and cfg["nu"] == pytest.approx(R / 500.0) and cfg["U"] == (0.0, 0.0, -1.0)
    g = wi.rng(12)
    for t in (math.pi / (2 * w), 3 * math.pi / (2 * w), 5 * math.pi / (2 * w)):
        A = 1 - np.array([1, 1, 0]) * 0.1 * math.cos(w * t)
        B = np.array([0, 0, 1]) * ((math.cos(w * t) - 1) * R / 4 - h)
        Cc = np.array([0, 0, 1]) * math.sin(w * t) * R / 4
        assert np.allclose(A, 1.0, atol=1e-15)
        for _ in range(40):
            x = np.array([g.uniform(0, n), g.uniform(0, n), g.uniform(0, 4 * n)])
            sphere = abs(math.sqrt(((A * x + B + Cc) ** 2).sum()) - R) - 1
            plane = (x + Cc)[2] - h
            assert wo.body_eval(cfg, x, t)[0] == pytest.approx(max(sphere, -plane), abs=1e-10)
    # and at a general time the zero level set is the listing's: points where the listing's sdf vanishes have d = 0
    t = 1.234
    A = 1 - np.array([1, 1, 0]) * 0.1 * math.cos(w * t)
    B = np.array([0, 0, 1]) * ((math.cos(w * t) - 1) * R / 4 - h)
    Cc = np.array([0, 0, 1]) * math.sin(w * t) * R / 4
    for _ in range(20):
        u = g.standard_normal(3); u[2] = abs(u[2]); u /= np.linalg.norm(u)
        xi = (R + 1.0) * u                                   # on the outer surface of the shell, in body coordinates
        x = (xi - B - Cc) / A
        if (x + Cc)[2] - h > 0.5:                            # clear of the cutting plane
            assert wo.body_eval(cfg, x, t)[0] == pytest.approx(0.0, abs=1e-10)


def test_shell_plane_and_sdf_arithmetic():
    base = dict(ndim=3, dims=(32, 32, 32), body_kind=wi.BODY_SPHERE, centre=(16.0, 16.0, 16.0), R=8.0)
    shell = wi.make(**base, shell=1.5)
    c = np.array(base["centre"])
    assert wo.body_eval(shell, c + [8, 0, 0], 0)[0] == pytest.approx(-1.5)            # on the mid-surface
    assert wo.body_eval(shell, c + [0, 9.5, 0], 0)[0] == pytest.approx(0.0, abs=1e-14)  # outer surface
    assert wo.body_eval(shell, c + [0, 0, 6.5], 0)[0] == pytest.approx(0.0, abs=1e-14)  # inner surface
    assert wo.body_eval(shell, c, 0)[0] == pytest.approx(8.0 - 1.5)                   # the hollow centre is OUTSIDE the body
    assert np.allclose(wo.body_eval(shell, c + [0, 0, 5.0], 0)[1], [0, 0, -1.0])        # inside the hollow the normal points inwards
    plane = wi.make(ndim=3, dims=(32, 32, 32), body_kind=wi.BODY_PLANE, centre=(0.0, 11.0, 0.0), axis=1)
    d, n, _ = wo.body_eval(plane, [3.0, 14.5, 7.0], 0)
    assert d == pytest.approx(3.5) and np.allclose(n, [0, 1, 0])
    # union and difference against the single primitives
    A = wi.make(**base)
    Bp = dict(kind=wi.BODY_SPHERE, centre=(22.0, 18.0, 16.0), R=5.0, motion=wi.MOTION_SIN, amp3=(0.0, 3.0, 0.0), freq3=(0.0, 0.05, 0.0), phase3=(0.0, 0.0, 0.0))
    B = wi.make(ndim=3, dims=(32, 32, 32), body_kind=wi.BODY_SPHERE, **{k: v for k, v in Bp.items() if k != "kind"})
    uni = wi.make(**base, parts=[dict(Bp, op="+")])
    dif = wi.make(**base, parts=[dict(Bp, op="-")])
    g = wi.rng(4)
    seen = set()
    for _ in range(300):
        x = c + g.uniform(-14, 14, 3)
        t = float(g.uniform(0, 20))
        dA, nA, vA = wo.body_eval(A, x, t)
        dB, nB, vB = wo.body_eval(B, x, t)
        dU, nU, vU = wo.body_eval(uni, x, t)
        dD, nD, vD = wo.body_eval(dif, x, t)
        assert dU == min(dA, dB) and dD == max(dA, -dB)
        assert np.array_equal(nU, nA if dA <= dB else nB) and np.array_equal(vU, vA if dA <= dB else vB)
        assert np.array_equal(nD, nA if dA >= -dB else -nB) and np.array_equal(vD, vA if dA >= -dB else vB)
        seen.add((dA <= dB, dA >= -dB))
    assert len(seen) >= 3                                     # every branch was exercised


def test_spin_gives_the_surface_speed_of_the_control_cylinder():
    """control circle of diameter d with scaled surface speed xi = d Omega / (2 U); V = Omega e_z x (x - c)."""
    D, xi = 32, 3.0
    cfg = wi.control_cylinders(D, xi=xi)
    small = cfg["parts"][0]
    d = 0.15 * D
    assert small["R"] == pytest.approx(d / 2) and abs(small["spin"]) * d / 2 == pytest.approx(xi)
    cs = np.array(small["centre"])
    big = np.array(cfg["centre"])
    assert np.linalg.norm(cs - big) == pytest.approx(D / 2 + 0.05 * D + d / 2)        # gap g/D = 0.05
    assert math.degrees(math.atan2(cs[1] - big[1], -(cs[0] - big[0]))) == pytest.approx(120.0)   # from the upstream direction
    for ang in np.linspace(0, 2 * math.pi, 7):
        x = cs + (d / 2 + 0.2) * np.array([math.cos(ang), math.sin(ang)])
        dd, n, v = wo.body_eval(cfg, x, 0.0)
        assert dd == pytest.approx(0.2, abs=1e-12)            # the small circle decides here
        assert abs(np.dot(v[:2], x - cs)) < 1e-12 and np.linalg.norm(v) == pytest.approx(abs(small["spin"]) * (d / 2 + 0.2))
        assert ((x - cs)[0] * v[1] - (x - cs)[1] * v[0]) * small["spin"] > 0    # sense of rotation
    # next to the big circle the body is at rest
    assert np.all(wo.body_eval(cfg, big + [-(D / 2 + 0.3), 0.0], 0.0)[2] == 0.0)


def test_measure_stores_the_composite_bodys_velocity_per_face():
    """measure! with a general body: V is a field (it is three scalars only for one rigid translation); mu0 and V at a few faces
    against body_eval + the kernel moments."""
    cfg = wi.jelly(3)
    o = wo.OracleSim(cfg)
    o.measure(2.5)
    V, mu0 = o.arr("V"), o.arr("mu0")
    g = wi.rng(5)
    assert np.ptp(V[2][mu0[2] < 1]) > 1e-3                    # not uniform
    for _ in range(50):
        i = int(g.integers(0, 3))
        c = [int(g.integers(2, n)) for n in cfg["dims"]]
        x = [c[0] - 0.5, c[1] - 0.5, c[2] - 0.5]
        x[i] -= 0.5
        d, n, v = wo.body_eval(cfg, x, 2.5)
        assert V[i][c[2], c[1], c[0]] == v[i]
        assert mu0[i][c[2], c[1], c[0]] == pytest.approx(wo.kernel_mu0(d, 1.0), abs=1e-15)
    o.close()
