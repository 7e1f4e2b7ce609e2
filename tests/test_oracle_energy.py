"""Pins for the oracle's kinetic-energy / enstrophy sums (reading R-E2; PAPER.md:169-173 follows the Taylor-Green vortex
by them) and for the half-domain Taylor-Green set-up between symmetry planes.  Closed forms of the
discrete sums, derived by hand for the staggered sampling of the vortex (s = sin(kappa/2)):
    sum_j sin^2(kappa j) = sum_j cos^2(kappa (j + 1/2)) = N/2 over one period (kappa = 2 pi/N) or half a period (pi/N);
    2-D:  KE = N^2/4,  w_z = 4 s sin(kappa x) sin(kappa y) at the cell corners  =>  Z = 2 s^2 N^2;
    3-D:  KE = N^3/8,  w_z as above times cos(kappa z), w_x = -2 s cos sin sin, w_y = -2 s sin cos sin  =>  Z = 3/2 s^2 N^3.
CPU only."""
import math

import numpy as np
import pytest

import wl_inputs as wi
from oracle import wl_oracle as wo


@pytest.mark.parametrize("n", [16, 64])
def test_energy_closed_forms_2d(n):
    s = wo.OracleSim(wi.tgv2d(n))
    s.init_tgv(1)
    ke, ens = s.energy()
    sk = math.sin(math.pi / n)                       # sin(kappa / 2), kappa = 2 pi / n
    assert ke == pytest.approx(n * n / 4.0, rel=1e-13)
    assert ens == pytest.approx(2.0 * sk * sk * n * n, rel=1e-12)
    # a uniform stream has no vorticity; KE counts every face once
    s.arr("u")[...] = 0.0
    s.arr("u")[0][...] = 3.0
    ke, ens = s.energy()
    assert ke == pytest.approx(0.5 * 9.0 * n * n) and ens == 0.0
    s.close()


@pytest.mark.parametrize("half", [False, True])
def test_energy_closed_forms_3d_full_and_half_domain(half):
    n = 16
    s = wo.OracleSim(wi.tgv3d_half(n) if half else wi.tgv3d(n))
    s.init_tgv(1)
    ke, ens = s.energy()
    sk = math.sin((math.pi / n if half else 2 * math.pi / n) / 2)
    assert ke == pytest.approx(n ** 3 / 8.0, rel=1e-13)
    assert ens == pytest.approx(1.5 * sk * sk * n ** 3, rel=1e-12)
    s.close()


def test_enstrophy_is_a_sum_of_squared_circulations():
    """brute force on a tiny 3-D field: the three circulations around the cell edges through the lower corner"""
    cfg = wi.make(ndim=3, dims=(6, 5, 4), periodic=(1, 0, 1), U=(0.0,) * 3)
    s = wo.OracleSim(cfg)
    s.set_fields(u=wi.random_velocity((6, 5, 4), seed=5, mean=(0.0, 0.0, 0.0)))
    u = s.arr("u")                                   # (3, S2, S1, S0) with BC-filled ghosts
    ke = ens = 0.0
    for z in range(1, 5):
        for y in range(1, 6):
            for x in range(1, 7):
                ke += 0.5 * sum(u[i, z, y, x] ** 2 for i in range(3))
                wz = (u[1, z, y, x] - u[1, z, y, x - 1]) - (u[0, z, y, x] - u[0, z, y - 1, x])
                wx = (u[2, z, y, x] - u[2, z, y - 1, x]) - (u[1, z, y, x] - u[1, z - 1, y, x])
                wy = (u[0, z, y, x] - u[0, z - 1, y, x]) - (u[2, z, y, x] - u[2, z, y, x - 1])
                ens += 0.5 * (wx * wx + wy * wy + wz * wz)
    assert np.allclose(s.energy(), [ke, ens], rtol=1e-13)
    s.close()


def test_half_domain_vortex_satisfies_the_symmetry_planes():
    """the half-domain between symmetry planes.  With kappa = pi/N the analytic vortex has zero normal
    velocity on every wall and even tangential components, so the slip-wall BC fill (R-M with U = 0) must leave the
    analytically sampled field -- ghosts included -- untouched, and the field is discretely divergence-free."""
    n = 12
    s = wo.OracleSim(wi.tgv3d_half(n))
    s.init_tgv(1)
    u = s.arr("u").copy()
    k = math.pi / n
    c = np.arange(n + 2) - 0.5                       # cell-centre coordinate of padded index 0..n+1
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    # (the normal component one cell OUTSIDE a wall, padded index 0, is set to U = 0 by R-M and read by nothing)
    assert np.allclose(u[0][:, :, 1:], (np.sin(k * (X - 0.5)) * np.cos(k * Y) * np.cos(k * Z))[:, :, 1:], atol=1e-14)
    assert np.allclose(u[1][:, 1:, :], (-np.cos(k * X) * np.sin(k * (Y - 0.5)) * np.cos(k * Z))[:, 1:, :], atol=1e-14)
    assert np.all(u[2] == 0.0)
    assert np.abs(u[0][:, :, 1]).max() < 1e-15 and np.abs(u[0][:, :, n + 1]).max() < 1e-15     # walls x = 0, pi
    assert np.abs(s.divergence()).max() < 1e-14
    s.close()


def test_2d_vortex_energy_and_enstrophy_decay_at_the_viscous_rate():
    """C1 (BASELINE configs[0]: 64^2, nu = dt = 0.01 physical, 20 steps): the 2-D Taylor-Green vortex is an exact
    solution whose amplitude decays as exp(-2 nu kappa^2 t), so KE and Z, both quadratic, decay as exp(-4 nu kappa^2 t)
    = exp(-0.008) -- with the DISCRETE Laplacian eigenvalue 2 (2 s)^2 in place of 2 kappa^2 (s = sin(kappa/2)), which at
    64 cells changes the exponent by 8e-4 relative.  The upwind-biased convective flux adds a little dissipation of its own
    (third-order: 2.4e-5 of the energy over these 20 steps), hence the tolerance 5e-5."""
    cfg = wi.baseline_config(0)
    s = wo.OracleSim(cfg)
    s.init_tgv(1)
    e0 = s.energy()
    for _ in range(20):
        s.mom_step(cfg["nu"])
    e1 = s.energy()
    n, nu = 64, cfg["nu"]
    rate = 2.0 * nu * 2.0 * (2.0 * math.sin(math.pi / n)) ** 2        # d/dt of a quadratic: twice the amplitude rate
    expect = math.exp(-rate * 20 * cfg["nu"])
    assert expect == pytest.approx(math.exp(-0.008), rel=1e-5)
    assert e1[0] / e0[0] == pytest.approx(expect, rel=5e-5)
    assert e1[1] / e0[1] == pytest.approx(expect, rel=5e-5)
    assert e1[0] / e0[0] < expect and e1[1] / e0[1] < expect          # the scheme never adds energy
    s.close()
