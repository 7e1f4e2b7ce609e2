"""Pins for the oracle's O1 (kernel moments), O2 (SDF / normal / body velocity / measure)
and the QUICK face value q(U,C,D) of O3 -- against quadrature, finite differences, closed
forms and hand-worked values (SURVEY.md 8(c) "What pins each part").  CPU only."""
import math

import numpy as np
import pytest
from scipy import integrate

import wl_inputs as wi
from golden_util import load
from oracle import wl_oracle as wo

G = load()


# ------------------------------------------------------------------ O1
@pytest.mark.parametrize("eps", [1.0, 2.0, 0.75])
def test_kernel_is_unit_mass_symmetric_compact(eps):
    m, _ = integrate.quad(lambda s: wo.kernel_K(s, eps), -eps, eps, epsabs=1e-13)
    assert abs(m - 1.0) < 1e-12
    assert wo.kernel_K(0.0, eps) == pytest.approx(1.0 / eps, abs=1e-15)
    assert wo.kernel_K(eps, eps) == 0.0 and wo.kernel_K(-1.5 * eps, eps) == 0.0
    for s in (0.1, 0.33, 0.9):
        assert wo.kernel_K(s * eps, eps) == pytest.approx(wo.kernel_K(-s * eps, eps), abs=1e-15)


@pytest.mark.parametrize("eps", [1.0, 2.0, 0.75])
def test_moments_match_quadrature(eps):
    """mu0(d) = int_{-eps}^{d} K, mu1(d) = int_{-d}^{eps} s K ds to 1e-9."""
    for a in np.linspace(-1.2, 1.2, 25):
        d = a * eps
        dc = min(max(d, -eps), eps)
        q0, _ = integrate.quad(lambda s: wo.kernel_K(s, eps), -eps, dc, epsabs=1e-13)
        q1, _ = integrate.quad(lambda s: s * wo.kernel_K(s, eps), -dc, eps, epsabs=1e-13)
        assert abs(wo.kernel_mu0(d, eps) - q0) < 1e-9
        assert abs(wo.kernel_mu1(d, eps) - q1) < 1e-9


def test_moment_special_values():
    for eps in (1.0, 2.5):
        assert wo.kernel_mu0(0.0, eps) == pytest.approx(G["mu0_at_0"], abs=1e-15)
        assert wo.kernel_mu0(eps, eps) == 1.0 and wo.kernel_mu0(-eps, eps) == 0.0
        assert wo.kernel_mu0(3 * eps, eps) == 1.0 and wo.kernel_mu0(-3 * eps, eps) == 0.0
        assert wo.kernel_mu1(0.0, eps) == pytest.approx(G["mu1_at_0_over_eps"] * eps, rel=1e-13)
        assert wo.kernel_mu1(eps, eps) == 0.0 and wo.kernel_mu1(-eps, eps) == 0.0
        # continuity at the edge of the band and mu0' = K
        assert abs(wo.kernel_mu1(0.999999 * eps, eps)) < 1e-9
        for d in (-0.7 * eps, 0.2 * eps):
            fd = (wo.kernel_mu0(d + 1e-6, eps) - wo.kernel_mu0(d - 1e-6, eps)) / 2e-6
            assert fd == pytest.approx(wo.kernel_K(d, eps), abs=1e-8)


# ------------------------------------------------------------------ O3: q(U,C,D)
def test_quick_hand_values():
    # cell averages of x^2 on [1,2],[2,3],[3,4] -> exact face value at 3 (SURVEY pins O3-iii)
    assert wo.quick(7 / 3, 19 / 3, 37 / 3) == pytest.approx(G["quick_quadratic_avg"], abs=1e-14)
    # same parabola mirrored: averages on [-2,-1],[-1,0],[0,1] = 7/3,1/3,1/3; the unlimited value
    # 0 lies outside [C,D] = {1/3}, so the limiter returns C
    assert wo.quick(7 / 3, 1 / 3, 1 / 3) == pytest.approx(1 / 3, abs=1e-15)
    # linear point data: face value midway between C and D
    assert wo.quick(0.0, 1.0, 2.0) == pytest.approx(1.5, abs=1e-15)
    assert wo.quick(2.0, 1.0, 0.0) == pytest.approx(0.5, abs=1e-15)
    # step: limiter returns C
    assert wo.quick(0.0, 0.0, 1.0) == 0.0
    # local extremum at C: reverts to first-order upwind value C
    assert wo.quick(0.0, 1.0, 0.0) == 1.0
    assert wo.quick(1.0, -2.0, 1.0) == -2.0


def test_quick_bounded_and_consistent():
    g = wi.rng(7)
    for _ in range(2000):
        U, Cc, D = g.uniform(-2, 2, 3)
        q = wo.quick(U, Cc, D)
        lo, hi = min(Cc, D), max(Cc, D)
        assert lo - 1e-15 <= q <= hi + 1e-15          # bounded by the two cells sharing the face
        # translation and scaling invariance of a median of affine expressions
        assert wo.quick(U + 3, Cc + 3, D + 3) == pytest.approx(q + 3, abs=1e-13)
        assert wo.quick(-2 * U, -2 * Cc, -2 * D) == pytest.approx(-2 * q, abs=1e-13)
    assert wo.quick(1.25, 1.25, 1.25) == 1.25


# ------------------------------------------------------------------ O2: SDF, normal, velocity
SPH = wi.make(ndim=3, dims=(32, 32, 32), body_kind=wi.BODY_SPHERE, centre=(16.0, 15.0, 17.0), R=8.0)
TOR = wi.make(ndim=3, dims=(48, 48, 48), body_kind=wi.BODY_TORUS, centre=(20.0, 24.0, 24.0), R=12.0, r=4.0, axis=0)
CIR = wi.make(ndim=2, dims=(32, 32), body_kind=wi.BODY_SPHERE, centre=(16.0, 16.0), R=6.0, periodic=(0, 0))
CYL = wi.make(ndim=3, dims=(32, 32, 8), body_kind=wi.BODY_CYLINDER, centre=(15.0, 17.0, 0.0), R=5.0, axis=2, periodic=(0, 0, 1))
CYLX = wi.make(ndim=3, dims=(8, 32, 32), body_kind=wi.BODY_CYLINDER, centre=(0.0, 15.0, 17.0), R=5.0, axis=0, periodic=(1, 0, 0))


def test_sdf_known_points():
    c = np.array(SPH["centre"])
    assert wo.body_eval(SPH, c, 0)[0] == pytest.approx(-8.0)
    assert wo.body_eval(SPH, c + [8, 0, 0], 0)[0] == pytest.approx(0.0, abs=1e-14)
    assert wo.body_eval(SPH, c + [0, 3, 4], 0)[0] == pytest.approx(-3.0)
    assert wo.body_eval(SPH, c + [0, 0, -20], 0)[0] == pytest.approx(12.0)
    t = np.array(TOR["centre"])
    assert wo.body_eval(TOR, t, 0)[0] == pytest.approx(12.0 - 4.0)                   # centre of the hole
    assert wo.body_eval(TOR, t + [0, 12, 0], 0)[0] == pytest.approx(-4.0)            # on the ring circle
    assert wo.body_eval(TOR, t + [0, 0, -12], 0)[0] == pytest.approx(-4.0)
    assert wo.body_eval(TOR, t + [5, 0, 0], 0)[0] == pytest.approx(13.0 - 4.0)       # on the axis: sqrt(144+25)
    assert wo.body_eval(TOR, t + [0, 16, 0], 0)[0] == pytest.approx(0.0, abs=1e-14)  # outer equator
    assert wo.body_eval(TOR, t + [3, 12, 0], 0)[0] == pytest.approx(-1.0)
    c2 = np.array(CIR["centre"])
    assert wo.body_eval(CIR, c2 + [3, 4], 0)[0] == pytest.approx(-1.0)


def test_cylinder_sdf_known_points_and_axis_invariance():
    """PAPER.md:121 'circular cylinder ... periodic boundary condition on the spanwise direction': d = distance from
    the axis - R, independent of the coordinate along the axis, normal in the cross-plane."""
    c = np.array(CYL["centre"])
    for z in (0.0, 3.3, 7.9, -40.0):
        assert wo.body_eval(CYL, c + [0, 0, z], 0)[0] == pytest.approx(-5.0)
        assert wo.body_eval(CYL, c + [3, 4, z], 0)[0] == pytest.approx(0.0, abs=1e-14)
        d, n, _ = wo.body_eval(CYL, c + [6, -8, z], 0)
        assert d == pytest.approx(5.0) and np.allclose(n, [0.6, -0.8, 0.0], atol=1e-15)
    cx = np.array(CYLX["centre"])
    d, n, _ = wo.body_eval(CYLX, cx + [2.5, 0, -13], 0)
    assert d == pytest.approx(8.0) and np.allclose(n, [0.0, 0.0, -1.0], atol=1e-15)


@pytest.mark.parametrize("cfg", [SPH, TOR, CIR, CYL, CYLX])
def test_normal_is_unit_gradient_of_sdf(cfg):
    g = wi.rng(11)
    nd = cfg["ndim"]
    h = 1e-5
    for _ in range(50):
        x = np.array(cfg["centre"][:nd]) + g.uniform(-14, 14, nd)
        d, n, _ = wo.body_eval(cfg, x, 0.0)
        fd = np.zeros(3)
        for k in range(nd):
            e = np.zeros(nd)
            e[k] = h
            fd[k] = (wo.body_eval(cfg, x + e, 0)[0] - wo.body_eval(cfg, x - e, 0)[0]) / (2 * h)
        assert np.allclose(n, fd, atol=1e-6)
        assert np.linalg.norm(n) == pytest.approx(1.0, abs=1e-12)


def test_heave_velocity_is_time_derivative_of_centre():
    cfg = wi.make(ndim=3, dims=(32, 32, 32), body_kind=wi.BODY_SPHERE, centre=(16.0, 16.0, 16.0), R=6.0,
                  motion=wi.MOTION_HEAVE_SIN, heave_dir=1, amp=3.0, freq=1 / 40.0, phase=0.3)
    x = np.array([16.0, 60.0, 16.0])                 # far above, on the heave axis: d = x_y - c_y - R
    cy = lambda t: x[1] - wo.body_eval(cfg, x, t)[0] - 6.0
    for t in (0.0, 3.7, 11.0, 25.0):
        assert cy(t) == pytest.approx(16.0 + 3.0 * math.sin(2 * math.pi * t / 40.0 + 0.3), abs=1e-12)
        _, _, v = wo.body_eval(cfg, x, t)
        fd = (cy(t + 1e-5) - cy(t - 1e-5)) / 2e-5
        assert v[1] == pytest.approx(fd, abs=1e-8)
        assert v[0] == 0.0 and v[2] == 0.0


def test_two_dof_motion_is_the_papers_map_and_V_its_time_derivative():
    """y = A_y sin(w t), x = A_x sin(2 w t + theta); V = dc/dt, uniform in space.  The centre is read
    back from the SDF at two far points on the axes through the initial centre."""
    D = 16.0
    cfg = wi.cylinder_2dof(16)
    Ax, Ay, th, w = 0.4 * D, 1.6 * D, math.pi / 6, 2 * math.pi / (5.4 * D)
    assert cfg["amp3"] == (Ax, Ay, 0.0) and cfg["phase3"] == (th, 0.0, 0.0)
    assert cfg["freq3"][0] == pytest.approx(2 * w / (2 * math.pi)) and cfg["freq3"][1] == pytest.approx(w / (2 * math.pi))
    c0 = np.array(cfg["centre"])
    far_x, far_y = c0 + [500.0, 0, 3.0], c0 + [0, 500.0, 5.0]

    def centre(t):
        # on the x axis through the moving centre d = |x - c_x| - R only if y = c_y: use Pythagoras on both probes
        dx = wo.body_eval(cfg, far_x, t)[0] + cfg["R"]          # sqrt((500 - ex)^2 + ey^2)
        dy = wo.body_eval(cfg, far_y, t)[0] + cfg["R"]          # sqrt(ex^2 + (500 - ey)^2)
        # two circles about the probes: solve for (ex, ey), the displacement of the centre
        # dx^2 - dy^2 = -1000 ex + 1000 ey  and  dx^2 = (500 - ex)^2 + ey^2
        k = (dx * dx - dy * dy) / 1000.0                         # ey - ex
        # (500 - ex)^2 + (ex + k)^2 = dx^2  ->  2 ex^2 + (2k - 1000) ex + 250000 + k^2 - dx^2 = 0, the small root
        a, b, cc = 2.0, 2 * k - 1000.0, 250000.0 + k * k - dx * dx
        ex = (-b - math.sqrt(b * b - 4 * a * cc)) / (2 * a)
        return np.array([ex, ex + k])

    for t in (0.0, 7.3, 21.0, 50.0, 86.4):
        e = centre(t)
        assert e[0] == pytest.approx(Ax * math.sin(2 * w * t + th), abs=1e-9)
        assert e[1] == pytest.approx(Ay * math.sin(w * t), abs=1e-9)
        _, _, v = wo.body_eval(cfg, c0 + [3.0, -2.0, 1.0], t)
        _, _, v2 = wo.body_eval(cfg, far_x, t)
        assert np.array_equal(v, v2)                              # rigid translation: V is uniform
        fd = (centre(t + 1e-4) - centre(t - 1e-4)) / 2e-4
        assert v[0] == pytest.approx(fd[0], abs=1e-6) and v[1] == pytest.approx(fd[1], abs=1e-6) and v[2] == 0.0
        assert v[0] == pytest.approx(2 * w * Ax * math.cos(2 * w * t + th), abs=1e-12)
        assert v[1] == pytest.approx(w * Ay * math.cos(w * t), abs=1e-12)
    # the motion closes after one period of the slow component, 5.4 D / U
    assert np.allclose(centre(5.4 * D), centre(0.0), atol=1e-9)


def test_cylinder_measure_is_invariant_along_the_axis_and_has_the_circle_area():
    """measure! of the spanning cylinder: every field is independent of z (the paper's periodic spanwise direction),
    and sum(1 - mu0) over the cells of one z-slab, with mu0 evaluated at the cell centres, is the area of the circle plus
    the kernel's second-moment correction: int (1 - mu0(|x| - R)) dA = pi (R^2 + s2)."""
    cfg = wi.make(ndim=3, dims=(32, 32, 8), body_kind=wi.BODY_CYLINDER, centre=(15.3, 16.6, 0.0), R=9.0, axis=2,
                  periodic=(0, 0, 1), U=(1.0, 0.0, 0.0))
    s = wo.OracleSim(cfg)
    for name in ("mu0", "mu1", "V", "iD"):
        a = s.interior(name)
        assert np.array_equal(a, np.broadcast_to(a[:, :1], a.shape)), name
    assert np.all(s.interior("mu1")[[2, 5, 8]] == 0.0)                # no normal component along the axis: mu1[i, z] = 0
    for l in range(1, s.nlevels):
        a = s.interior("L", l)
        assert np.array_equal(a, np.broadcast_to(a[:, :1], a.shape))
    s.close()
    s2 = 1 / 3 - 2 / math.pi ** 2
    area = 0.0
    for x in np.arange(32) + 0.5:
        for y in np.arange(32) + 0.5:
            d = wo.body_eval(cfg, [x, y, 0.5], 0.0)[0]
            area += 1.0 - wo.kernel_mu0(d, 1.0)
    assert area == pytest.approx(math.pi * (81.0 + s2), rel=1e-3)


def _centre_mu0_volume(cfg):
    """sum over cells of (1 - mu0(d at the cell centre)): uses body_eval + kernel_mu0 only."""
    nd = cfg["ndim"]
    dims = cfg["dims"][:nd]
    vol = 0.0
    axes = [np.arange(n) + 0.5 for n in dims]
    pts = np.stack(np.meshgrid(*axes, indexing="ij"), -1).reshape(-1, nd)
    for x in pts:
        d = wo.body_eval(cfg, x, 0.0)[0]
        if d < cfg["eps"]:
            vol += 1.0 - wo.kernel_mu0(d, cfg["eps"])
    return vol


def test_body_volume_from_mu0():
    """sum(1 - mu0(d)) -> body volume + the kernel's second-moment correction (closed form):
    int (1-mu0(|x|-R)) dV = 4pi/3 int K(s)(R+s)^3 ds = 4/3 pi R^3 + 4 pi R s2, and by Pappus
    2 pi^2 R (r^2 + s2) for the torus, with s2 = int s^2 K ds (odd moments vanish)."""
    s2, _ = integrate.quad(lambda s: s * s * wo.kernel_K(s, 1.0), -1, 1, epsabs=1e-13)
    assert s2 == pytest.approx(1 / 3 - 2 / math.pi ** 2, abs=1e-12)
    sph = wi.make(ndim=3, dims=(24, 24, 24), body_kind=wi.BODY_SPHERE, centre=(12.0, 12.0, 12.0), R=8.0)
    tor = wi.make(ndim=3, dims=(12, 36, 36), body_kind=wi.BODY_TORUS, centre=(6.0, 18.0, 18.0), R=12.0, r=4.0)
    assert _centre_mu0_volume(sph) == pytest.approx(G["sphere_volume_R8"] + 4 * math.pi * 8.0 * s2, rel=1e-3)
    assert _centre_mu0_volume(tor) == pytest.approx(G["torus_volume_R12_r4"] + 2 * math.pi ** 2 * 12.0 * s2, rel=1e-3)


def test_measure_fields_sphere():
    """measure(): staggered sampling position, mu1 = mu1(d) n, domain rule, mirror symmetry."""
    cfg = wi.sphere((32, 24, 24), D=10.0, centre=(12.0, 12.0, 12.0))
    s = wo.OracleSim(cfg)
    mu0, mu1, V = s.arr("mu0"), s.arr("mu1"), s.arr("V")
    # sample faces: component i at (c - 1/2) - e_i/2   (c = padded C index)
    g = wi.rng(3)
    for _ in range(200):
        c = np.array([g.integers(2, 33), g.integers(2, 25), g.integers(2, 25)])   # off the zeroed boundary faces
        for i in range(3):
            xf = c - 0.5
            xf[i] -= 0.5
            d, n, v = wo.body_eval(cfg, xf, 0.0)
            if i == 0 and c[0] == 1:
                continue
            assert mu0[i, c[2], c[1], c[0]] == pytest.approx(wo.kernel_mu0(d, 1.0), abs=1e-15)
            for j in range(3):
                assert mu1[i * 3 + j, c[2], c[1], c[0]] == pytest.approx(wo.kernel_mu1(d, 1.0) * n[j], abs=1e-15)
    assert np.all(V == 0.0)
    # domain rule: mu0 = 0 on boundary-normal faces (c_j = 1 and N_j+1), non-periodic
    assert np.all(mu0[0, :, :, 1] == 0) and np.all(mu0[0, :, :, 33] == 0)
    assert np.all(mu0[1, :, 1, :] == 0) and np.all(mu0[1, :, 25, :] == 0)
    assert np.all(mu0[2, 1, :, :] == 0) and np.all(mu0[2, 25, :, :] == 0)
    # mirror symmetry about the body centre planes y = 12, z = 12 (x-face field, interior)
    a = mu0[0, 1:-1, 1:-1, 1:-1]
    assert np.array_equal(a, a[:, ::-1, :]) and np.array_equal(a, a[::-1, :, :])
    # deep inside the body mu0 = 0, far away mu0 = 1, mu1 = 0 in both
    assert mu0[1, 12, 12, 12] == 0.0 and mu0[1, 12, 12, 28] == 1.0
    assert np.all(mu1[:, 12, 12, 28] == 0.0)
    s.close()


def test_measure_no_body_and_periodic_wrap():
    s = wo.OracleSim(wi.tgv2d(16))
    assert np.all(s.arr("mu0") == 1.0) and np.all(s.arr("mu1") == 0.0) and np.all(s.arr("V") == 0.0)
    s.close()
    # heaving body: V uniform = dc/dt wherever measured; periodic z ghosts wrapped
    cfg = wi.heaving_sphere((24, 24, 16), D=8.0, centre=(10.0, 12.0, 8.0), periodic=(0, 0, 1))
    s = wo.OracleSim(cfg)
    s.measure(7.5)
    V = s.arr("V")
    vy = cfg["amp"] * 2 * math.pi * cfg["freq"] * math.cos(2 * math.pi * cfg["freq"] * 7.5)
    assert np.allclose(V[1], vy, atol=1e-15) and np.all(V[0] == 0) and np.all(V[2] == 0)
    mu0 = s.arr("mu0")
    assert np.array_equal(mu0[:, 0], mu0[:, 16]) and np.array_equal(mu0[:, 17], mu0[:, 1])
    s.close()
