"""Pins for the oracle's O3 (conv_diff), O4 (BDIM blend), O5 (BC fill), O6 (convective
exit): invariants, special cases that reduce to textbook operators, hand-worked values and
a convergence-order check against an analytically differentiated field.  CPU only."""
import math

import numpy as np
import pytest

import wl_inputs as wi
from oracle import wl_oracle as wo


def _sim(**kw):
    return wo.OracleSim(wi.make(**kw))


# ------------------------------------------------------------------ O3
@pytest.mark.parametrize("per", [(1, 1, 1), (0, 0, 0), (0, 1, 0)])
def test_uniform_flow_has_zero_rhs(per):
    s = _sim(ndim=3, dims=(12, 10, 8), U=(1.0, -0.5, 0.25), nu=0.3, periodic=per)
    for i, v in enumerate((1.0, -0.5, 0.25)):
        s.arr("u")[i][...] = v
    s.conv_diff("u")
    assert np.all(s.interior("f") == 0.0)
    s.close()


@pytest.mark.parametrize("dims", [(16, 12), (12, 10, 8)])
def test_periodic_rhs_sums_to_zero(dims):
    """Conservative form: on a periodic box the fluxes telescope, sum_c r_i[c] = 0."""
    nd = len(dims)
    s = _sim(ndim=nd, dims=dims, periodic=(1,) * nd, nu=0.05, U=(0.0,) * 3)
    s.set_fields(u=wi.random_velocity(dims))
    s.conv_diff("u")
    r = s.interior("f")
    for i in range(nd):
        assert abs(r[i].sum()) < 1e-11 * np.abs(r[i]).sum()
    s.close()


@pytest.mark.parametrize("dims", [(16, 12), (10, 8, 6)])
def test_diffusion_term_is_textbook_laplacian(dims):
    """r(nu=1) - r(nu=0) on a periodic box is the 5/7-point Laplacian (np.roll stencil)."""
    nd = len(dims)
    u = wi.random_velocity(dims, seed=5)
    out = []
    for nu in (0.0, 1.0):
        s = _sim(ndim=nd, dims=dims, periodic=(1,) * nd, nu=nu, U=(0.0,) * 3)
        s.set_fields(u=u)
        s.conv_diff("u")
        out.append(s.interior("f").copy().reshape(u.shape))
        s.close()
    lap = np.zeros_like(u)
    for ax in range(1, nd + 1):
        lap += np.roll(u, 1, axis=ax) + np.roll(u, -1, axis=ax) - 2 * u
    assert np.allclose(out[1] - out[0], lap, atol=1e-12)


def test_diffusion_term_nonperiodic_uses_ghosts():
    """Non-periodic: the same Laplacian taken on the BC-filled padded array (np.pad-free)."""
    dims = (10, 8)
    u = wi.random_velocity(dims, seed=6)
    res = []
    for nu in (0.0, 1.0):
        s = _sim(ndim=2, dims=dims, periodic=(0, 0), nu=nu, U=(1.0, 0.0, 0.0))
        s.set_fields(u=u)
        up = s.arr("u").copy()
        s.conv_diff("u")
        res.append(s.interior("f").copy())
        s.close()
    a = up[:, 0]
    lap = (a[:, 1:-1, :-2] + a[:, 1:-1, 2:] + a[:, :-2, 1:-1] + a[:, 2:, 1:-1] - 4 * a[:, 1:-1, 1:-1])
    assert np.allclose((res[1] - res[0])[:, 0], lap, atol=1e-12)


def test_convective_flux_hand_example_1d_like():
    """2-D field depending on x only, v = 0, nu = 0, u > 0 monotone-linear: the face value is
    the midpoint (QUICK exact on linear point data), so r_x = -(F_e - F_w) with
    F = phi*psi = ((u_c+u_m)/2)^2 evaluated by hand."""
    dims = (12, 6)
    s = _sim(ndim=2, dims=dims, periodic=(0, 1), nu=0.0, U=(1.0, 0.0, 0.0))
    up = s.arr("u")
    xs = np.arange(14) - 1.0                      # face position of u_x[c] is c-1
    up[0][0, :, :] = (1.0 + 0.1 * xs)[None, :]
    up[1][...] = 0.0
    s.conv_diff("u")
    r = s.interior("f")[0, 0]
    uf = 1.0 + 0.1 * xs
    # flux through the lower x-boundary of the CV of u_x[c] (at the centre of cell c-1)
    F = lambda c: (0.5 * (uf[c - 1] + uf[c])) ** 2
    for c in range(2, 12):                        # away from the boundary fallback planes
        assert r[3, c - 1] == pytest.approx(F(c) - F(c + 1), abs=1e-14)
    # r_y = 0: v = 0 everywhere
    assert np.all(s.interior("f")[1] == 0.0)
    s.close()


def test_upwind_direction_follows_sign_of_phi():
    """A unit step in the passive component v (0 for i<8, 1 for i>=8, periodic, 16 cells)
    advected by u = +1 or -1, nu = 0.  Worked by hand with q(U,C,D): the limited face value
    is the upwind cell at both discontinuities, so with u=+1 the x-flux u*psi is 0 at faces
    i<=8 and 1 at faces 9..16(=0)  =>  r_v = F(i)-F(i+1) = -1 at i=8, +1 at i=0, else 0;
    with u=-1 the flux is -1 at faces 8..15 and 0 elsewhere  =>  r_v = +1 at i=7, -1 at i=15."""
    dims = (16, 8)
    for sign, expect in ((+1.0, {8: -1.0, 0: 1.0}), (-1.0, {7: 1.0, 15: -1.0})):
        s = _sim(ndim=2, dims=dims, periodic=(1, 1), nu=0.0, U=(0.0, 0.0, 0.0))
        u = np.zeros((2, 8, 16))
        u[0] = sign
        u[1][:, 8:] = 1.0
        s.set_fields(u=u)
        s.conv_diff("u")
        rv = s.interior("f")[1, 0, 4]
        want = np.zeros(16)
        for k, v in expect.items():
            want[k] = v
        assert np.allclose(rv, want, atol=1e-14)
        assert np.all(s.interior("f")[0] == 0.0)
        s.close()


def test_convergence_order_against_analytic_rhs():
    """r -> -d_j(u_j u_i) + nu lap u_i at second order on a smooth periodic field with a mean
    stream (error ratio ~4 per refinement in the mean-abs norm; the limiter only clips at
    isolated extrema).  The target is differentiated by hand, independently of the oracle."""
    nu = 0.7
    errs = []
    for n in (16, 32, 64):
        k = 2 * math.pi / n
        s = _sim(ndim=2, dims=(n, n), periodic=(1, 1), nu=nu, U=(0.0, 0.0, 0.0))
        j, i = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")     # j = y index, i = x index
        A, U0, V0 = 0.3, 1.0, 0.6
        fu = lambda x, y: U0 + A * np.sin(k * x) * np.cos(k * y)
        fv = lambda x, y: V0 - A * np.cos(k * x) * np.sin(k * y)
        xu, yu = i.astype(float), j + 0.5          # x-face of cell (C index i+1): x = i, y = j+1/2
        xv, yv = i + 0.5, j.astype(float)
        s.set_fields(u=np.stack([fu(xu, yu), fv(xv, yv)]))
        s.conv_diff("u")
        r = s.interior("f")[:, 0]

        def exact(x, y, comp):
            u, v = fu(x, y), fv(x, y)
            ux, uy = A * k * np.cos(k * x) * np.cos(k * y), -A * k * np.sin(k * x) * np.sin(k * y)
            vx, vy = A * k * np.sin(k * x) * np.sin(k * y), -A * k * np.cos(k * x) * np.cos(k * y)
            if comp == 0:
                return -(2 * u * ux + vy * u + v * uy) + nu * (-2 * k * k) * (u - U0)
            return -(ux * v + u * vx + 2 * v * vy) + nu * (-2 * k * k) * (v - V0)

        e = np.abs(r[0] - exact(xu, yu, 0)).mean() + np.abs(r[1] - exact(xv, yv, 1)).mean()
        errs.append(e * n)                         # scale out the k ~ 1/n amplitude of the target
        s.close()
    assert errs[0] / errs[1] > 3.3 and errs[1] / errs[2] > 3.3


def test_boundary_fallback_is_central_average():
    """Non-periodic lower plane with phi > 0: psi = (w[c-1]+w[c])/2 (reading R-H).  Checked on
    the y-flux of u_x through the bottom wall plane with a constant positive v."""
    dims = (8, 6)
    g = wi.rng(9)
    # x-independent field, so the x-fluxes cancel and only the y-fluxes of u_x remain
    s = _sim(ndim=2, dims=dims, periodic=(1, 0), nu=0.0, U=(0.0, 0.0, 0.0))
    up = s.arr("u")
    col = g.uniform(1, 2, 8)
    up[0][0, :, :] = col[:, None]
    up[1][...] = 0.5
    s.conv_diff("u")
    r = s.interior("f")[0, 0]
    lo = 0.5 * 0.5 * (col[0] + col[1])
    hi = 0.5 * wo.quick(col[0], col[1], col[2])
    assert r[0, 3] == pytest.approx(lo - hi, abs=1e-14)
    s.close()


# ------------------------------------------------------------------ O4
def test_bdim_identity_without_body():
    dims = (10, 8, 6)
    s = _sim(ndim=3, dims=dims, periodic=(1, 1, 1), nu=0.1, U=(0.0,) * 3)
    s.set_fields(u=wi.random_velocity(dims))
    s.arr("u0")[...] = s.arr("u")
    s.conv_diff("u0")
    r = s.interior("f").copy()
    dt = 0.37
    s.bdim(dt, 0)
    assert np.allclose(s.interior("u"), s.interior("u0") + dt * r, atol=1e-15)
    # corrector form: (u' + B)/2
    uprime = s.interior("u").copy()
    s.conv_diff("u")
    r2 = s.interior("f").copy()
    s.bdim(dt, 1)
    assert np.allclose(s.interior("u"), 0.5 * (uprime + s.interior("u0") + dt * r2), atol=1e-15)
    s.close()


def test_bdim_solid_takes_body_velocity_and_mu1_indexing():
    """mu0 = 0, mu1 = 0 => u = V.  Then constant mu0 = m, mu1[i,j] = M[i][j], linear f:
    u_i = V_i + m f_i + sum_j M[i][j] G[i][j] -- fails if mu1 is indexed transposed."""
    dims = (8, 7, 6)
    s = _sim(ndim=3, dims=dims, periodic=(0, 0, 0), nu=0.0, U=(0.0,) * 3)
    g = wi.rng(4)
    s.arr("mu0")[...] = 0.0
    s.arr("mu1")[...] = 0.0
    s.arr("V")[...] = g.uniform(-1, 1, s.arr("V").shape)
    s.arr("u0")[...] = g.uniform(-1, 1, s.arr("u0").shape)
    s.arr("f")[...] = 0.0
    s.bdim(0.5, 0)
    assert np.array_equal(s.interior("u"), s.interior("V"))
    M = g.uniform(-1, 1, (3, 3))
    Gm = g.uniform(-1, 1, (3, 3))
    a0 = g.uniform(-1, 1, 3)
    Sz, Sy, Sx = s.arr("p").shape[1:]
    zz, yy, xx = np.meshgrid(np.arange(Sz), np.arange(Sy), np.arange(Sx), indexing="ij")
    for i in range(3):
        s.arr("u0")[i][...] = a0[i] + Gm[i, 0] * xx + Gm[i, 1] * yy + Gm[i, 2] * zz
        for j in range(3):
            s.arr("mu1")[i * 3 + j][...] = M[i, j]
    s.arr("mu0")[...] = 0.3
    s.arr("V")[...] = 0.0
    s.arr("f")[...] = 0.0                          # r = 0
    s.bdim(0.5, 0)
    for i in range(3):
        expect = 0.3 * s.interior("u0")[i] + (M[i] * Gm[i]).sum()
        assert np.allclose(s.interior("u")[i], expect, atol=1e-13)
    s.close()


# ------------------------------------------------------------------ O5 / O6
def test_bc_fill_identities():
    dims = (8, 6, 5)
    s = _sim(ndim=3, dims=dims, periodic=(0, 0, 1), exit_bc=1, U=(1.0, 0.2, 0.0))
    g = wi.rng(2)
    s.arr("u")[...] = g.uniform(-1, 1, s.arr("u").shape)
    before = s.arr("u").copy()
    s.bc()
    u = s.arr("u")
    # interior untouched except the prescribed normal faces
    assert np.array_equal(u[1:, 1:-1, 2:-1, 1:-1][:1], before[1:, 1:-1, 2:-1, 1:-1][:1])
    # x: inflow normal at c=0,1 ; exit plane (c=9) untouched on the interior of the other directions
    assert np.all(u[0, :, :, 0] == 1.0) and np.all(u[0, :, :, 1] == 1.0)
    assert np.array_equal(u[0, 1:-1, 1:-1, 9], before[0, 1:-1, 1:-1, 9])
    # x: tangential slip ghosts
    assert np.array_equal(u[1, 1:-1, 2:-1, 0], u[1, 1:-1, 2:-1, 1])
    assert np.array_equal(u[2, 1:-1, 1:-1, 9], u[2, 1:-1, 1:-1, 8])
    # y: normal = U_y on c=0,1,N+1 ; tangential copy
    assert np.all(u[1, :, 0, :] == 0.2) and np.all(u[1, :, 1, :] == 0.2) and np.all(u[1, :, 7, :] == 0.2)
    assert np.array_equal(u[0, 1:-1, 0, :], u[0, 1:-1, 1, :]) and np.array_equal(u[0, 1:-1, 7, :], u[0, 1:-1, 6, :])
    # z periodic: all components wrap
    assert np.array_equal(u[:, 0], u[:, 5]) and np.array_equal(u[:, 6], u[:, 1])
    s.close()


def test_exit_bc_mass_balance_and_upwind_formula():
    dims = (8, 6, 5)
    s = _sim(ndim=3, dims=dims, periodic=(0, 0, 0), exit_bc=1, U=(1.0, 0.0, 0.0))
    g = wi.rng(12)
    s.arr("u0")[...] = g.uniform(0.5, 1.5, s.arr("u0").shape)
    s.arr("u")[...] = 123.0
    dt = 0.4
    u0 = s.arr("u0")[0]
    raw = u0[1:-1, 1:-1, 9] - 1.0 * dt * (u0[1:-1, 1:-1, 9] - u0[1:-1, 1:-1, 8])
    s.exit_bc(dt)
    ex = s.arr("u")[0][1:-1, 1:-1, 9]
    assert ex.sum() == pytest.approx(1.0 * ex.size, abs=1e-12)
    assert np.allclose(ex, raw - (raw.mean() - 1.0), atol=1e-14)
    # everything else untouched
    assert np.all(s.arr("u")[0][:, :, :9] == 123.0) and np.all(s.arr("u")[1:] == 123.0)
    # a uniform stream passes unchanged
    s.arr("u0")[...] = 1.0
    s.arr("u")[...] = 1.0
    s.exit_bc(dt)
    assert np.all(s.arr("u")[0] == 1.0)
    s.close()
