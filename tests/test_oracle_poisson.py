"""Pins for the oracle's O7 (Poisson operator, project) and O8 (multigrid + PCG smoother):
textbook Laplacians built with scipy.sparse kron, symmetry / null-space invariants, the
dense direct solve on 16x16 named in BASELINE.json north_star, coarse-operator
consistency, monotone residual decrease and divergence after projection.  CPU only."""
import numpy as np
import pytest
import scipy.sparse as sp

import wl_inputs as wi
from oracle import wl_oracle as wo


def _pad(a):
    return np.pad(a, [(0, 0)] + [(1, 1)] * (a.ndim - 1)) if a.ndim == 3 else np.pad(a, 1)


def _apply(s, level, x_int):
    """q = A_level x for an interior-shaped x ([Nz,]Ny,Nx) -> interior-shaped q."""
    shp = s.arr("x", level).shape[1:]
    xp = np.zeros(shp)
    if s.nd == 3:
        xp[1:-1, 1:-1, 1:-1] = x_int
    else:
        xp[0, 1:-1, 1:-1] = x_int
    q, d = s.matvec(level, xp)
    return (q[1:-1, 1:-1, 1:-1] if s.nd == 3 else q[0, 1:-1, 1:-1]), d


def _lap1d(n, periodic):
    T = sp.diags([np.ones(n - 1), -2 * np.ones(n), np.ones(n - 1)], [-1, 0, 1]).tolil()
    if periodic:
        T[0, n - 1] = 1
        T[n - 1, 0] = 1
    else:                      # homogeneous Neumann: boundary faces carry no flux
        T[0, 0] = -1
        T[n - 1, n - 1] = -1
    return T.tocsr()


@pytest.mark.parametrize("dims,per", [((12, 10), (1, 1)), ((12, 10), (0, 0)), ((8, 6, 10), (1, 0, 1)),
                                      ((8, 6, 10), (0, 0, 0))])
def test_operator_is_textbook_laplacian_without_body(dims, per):
    nd = len(dims)
    s = wo.OracleSim(wi.make(ndim=nd, dims=dims, periodic=per, U=(0.0,) * 3))
    x = wi.random_scalar(dims, seed=3)
    q, _ = _apply(s, 0, x)
    # kron sum, x fastest: A = I (x) I (x) Tx + I (x) Ty (x) I + Tz (x) I (x) I
    Ts = [_lap1d(dims[d], per[d]) for d in range(nd)]
    eye = [sp.identity(dims[d]) for d in range(nd)]
    A = None
    for d in range(nd):
        mats = [Ts[k] if k == d else eye[k] for k in reversed(range(nd))]
        term = mats[0]
        for m in mats[1:]:
            term = sp.kron(term, m)
        A = term if A is None else A + term
    assert np.allclose(q.ravel(), A @ x.ravel(), atol=1e-12)
    s.close()


def _body_sims():
    yield wo.OracleSim(wi.make(ndim=2, dims=(16, 16), periodic=(0, 0), body_kind=wi.BODY_SPHERE,
                               centre=(7.3, 8.1), R=3.4, U=(1.0, 0, 0)))
    yield wo.OracleSim(wi.sphere((16, 12, 12), D=6.0, centre=(6.0, 6.0, 6.0)))
    yield wo.OracleSim(wi.make(ndim=3, dims=(16, 8, 8), periodic=(0, 1, 1), body_kind=wi.BODY_SPHERE,
                               centre=(6.0, 4.0, 4.0), R=2.5))


def test_operator_symmetric_nullspace_all_levels():
    g = wi.rng(21)
    for s in _body_sims():
        for lev in range(s.nlevels):
            shp = s.interior("x", lev).shape[1:] if s.nd == 3 else s.interior("x", lev).shape[2:]
            x, y = g.standard_normal(shp), g.standard_normal(shp)
            Ax, _ = _apply(s, lev, x)
            Ay, _ = _apply(s, lev, y)
            assert (y * Ax).sum() == pytest.approx((x * Ay).sum(), rel=1e-11, abs=1e-11)
            A1, _ = _apply(s, lev, np.ones(shp))
            assert np.abs(A1).max() < 1e-13
            assert (x * Ax).sum() <= 1e-12            # negative semi-definite
            # diagonal: iD = 1/D with D = (A e_c)_c, checked on a few cells by brute force
            iD = s.interior("iD", lev)[0] if s.nd == 3 else s.interior("iD", lev)[0, 0]
            for _ in range(5):
                c = tuple(int(g.integers(0, n)) for n in shp)
                e = np.zeros(shp)
                e[c] = 1.0
                D = _apply(s, lev, e)[0][c]
                assert iD[c] == pytest.approx(1.0 / D if D != 0 else 0.0, rel=1e-13)
        s.close()


def test_coarse_coefficients_uniform():
    """L == 1 on the fine level => coarse L = 1 in 2-D and 2 in 3-D (1/2 * 2^(n-1))."""
    s = wo.OracleSim(wi.tgv2d(32, max_levels=0))
    for lev in range(1, s.nlevels):
        assert np.all(s.interior("L", lev) == 1.0)
    s.close()
    s = wo.OracleSim(wi.tgv3d(16))
    assert s.nlevels == 3
    assert np.all(s.interior("L", 1) == 2.0) and np.all(s.interior("L", 2) == 4.0)
    s.close()


def test_hierarchy_rule_matches_survey():
    """C1 4 levels (cap), C2 6 to 4^3, C3 6 to 8x4x4, C4 7 to 8x4x4, C5 7 to 6x4x4.
    Checked with the rule alone (no allocation of the big grids)."""
    def levels(dims, cap=0):
        n, k = list(dims), 1
        while (cap <= 0 or k < cap) and all(v % 2 == 0 and v > 4 for v in n):
            n = [v // 2 for v in n]
            k += 1
        return k, tuple(n)
    assert levels((64, 64), 4) == (4, (8, 8))
    assert levels((128,) * 3) == (6, (4, 4, 4))
    assert levels((256, 128, 128)) == (6, (8, 4, 4))
    assert levels((512, 256, 256)) == (7, (8, 4, 4))
    assert levels((384, 256, 256)) == (7, (6, 4, 4))
    for k, scale in ((0, 1), (1, 4), (2, 4), (4, 8)):
        cfg = wi.baseline_config(k, scale)
        s = wo.OracleSim(cfg)
        assert s.nlevels == levels(cfg["dims"][: cfg["ndim"]], cfg["max_levels"])[0]
        s.close()


def _dense(s):
    n = int(np.prod(s.dims))
    shp = tuple(reversed(s.dims))
    A = np.zeros((n, n))
    for k in range(n):
        e = np.zeros(n)
        e[k] = 1.0
        A[:, k] = _apply(s, 0, e.reshape(shp))[0].ravel()
    return A


def test_multigrid_matches_dense_direct_solve_16x16():
    """BASELINE north_star pin: MG pressure == dense direct solve on a 16x16 grid with a
    circular body (variable coefficients).  x is defined up to a constant per connected
    fluid region (reading R-P): compare the mean-free solution over cells with D != 0."""
    cfg = wi.make(ndim=2, dims=(16, 16), periodic=(0, 0), body_kind=wi.BODY_SPHERE, centre=(7.3, 8.1), R=3.4,
                  U=(1.0, 0, 0), fixed_vcycles=0, tol=1e-12, max_vcycles=200)
    s = wo.OracleSim(cfg)
    assert s.nlevels == 3
    A = _dense(s)
    assert np.allclose(A, A.T, atol=1e-14)
    live = np.abs(np.diag(A)) > 0
    g = wi.rng(5)
    z = g.standard_normal(256)
    z[~live] = 0.0
    z[live] -= z[live].mean()                       # compatible right-hand side
    xd = np.linalg.lstsq(A[np.ix_(live, live)], z[live], rcond=None)[0]
    s.interior("sig")[0, 0][...] = z.reshape(16, 16)
    s.arr("x")[...] = 0.0
    nv = s.solve()
    xm = s.interior("x")[0, 0].ravel()[live]
    assert nv < 60
    assert np.abs(A[np.ix_(live, live)] @ xd - z[live]).max() < 1e-10
    assert np.allclose(xm - xm.mean(), xd - xd.mean(), atol=1e-9)
    s.close()


def test_multigrid_matches_sparse_direct_solve_3d_periodic():
    cfg = wi.make(ndim=3, dims=(16, 8, 8), periodic=(0, 1, 1), body_kind=wi.BODY_SPHERE, centre=(6.0, 4.0, 4.0),
                  R=2.5, fixed_vcycles=0, tol=1e-12, max_vcycles=200)
    s = wo.OracleSim(cfg)
    A = _dense(s)
    live = np.abs(np.diag(A)) > 0
    z = wi.rng(6).standard_normal(A.shape[0])
    z[~live] = 0
    z[live] -= z[live].mean()
    xd = np.linalg.lstsq(A[np.ix_(live, live)], z[live], rcond=None)[0]
    s.interior("sig")[0][...] = z.reshape(8, 8, 16)
    s.arr("x")[...] = 0.0
    s.solve()
    xm = s.interior("x")[0].ravel()[live]
    assert np.allclose(xm - xm.mean(), xd - xd.mean(), atol=1e-9)
    s.close()


def test_residual_decreases_every_vcycle_and_pcg_alone_converges():
    cfg = wi.sphere((32, 16, 16), D=8.0, centre=(8.0, 8.0, 8.0))
    s = wo.OracleSim(cfg)
    live = s.interior("iD")[0] != 0
    z = wi.random_scalar((32, 16, 16), seed=8)
    z[~live] = 0
    z[live] -= z[live].mean()
    s.interior("sig")[0][...] = z
    s.arr("x")[...] = 0.0
    s.residual()
    hist = [np.abs(s.interior("r")).max()]
    for _ in range(8):
        s.vcycle(0)
        s.smooth(0, cfg["smooth_iters"])
        hist.append(np.abs(s.interior("r")).max())
    assert all(b < 0.5 * a for a, b in zip(hist, hist[1:]))
    assert hist[-1] < 1e-6 * hist[0]
    # r always equals z - A x (the increments keep it consistent)
    r_saved = s.interior("r").copy()
    s.residual()
    assert np.allclose(s.interior("r"), r_saved, atol=1e-12)
    # PCG alone (no coarse grids) is a convergent iteration: energy norm decreases
    s.arr("x")[...] = 0.0
    s.residual()
    r0 = np.linalg.norm(s.interior("r"))
    s.smooth(0, 200)                       # one call stops after a 1e-4 reduction (R-T, theta)
    assert np.linalg.norm(s.interior("r")) < 1e-3 * r0
    s.smooth(0, 200)                       # restarted calls keep converging
    s.smooth(0, 200)
    assert np.linalg.norm(s.interior("r")) < 1e-6 * r0
    s.close()


def test_pcg_exact_in_n_steps_on_tiny_system():
    """CG terminates in at most (#distinct non-zero eigenvalues) steps: 4x4 periodic Laplacian
    has eigenvalues {-2,-4,-6,-8} (+0), so 4 iterations solve any compatible system."""
    s = wo.OracleSim(wi.make(ndim=2, dims=(4, 4), periodic=(1, 1), U=(0.0,) * 3))
    z = wi.rng(1).standard_normal((4, 4))
    z -= z.mean()
    s.interior("sig")[0, 0][...] = z
    s.arr("x")[...] = 0.0
    s.residual()
    s.smooth(0, 4)
    assert np.abs(s.interior("r")).max() < 1e-13
    s.close()


def test_smoother_guards():
    s = wo.OracleSim(wi.tgv2d(8, max_levels=1))
    s.arr("x")[...] = 0.0
    s.arr("sig")[...] = 0.0
    s.residual()
    s.smooth(0, 6)                                   # rho = 0 -> immediate return
    assert np.all(s.arr("x") == 0.0) and np.all(np.isfinite(s.arr("r")))
    s.close()


def test_smoother_removes_the_incompatible_part_of_the_residual():
    """R-T2: constants span the null space of A (per coupled region; buried cells are decoupled), so the
    smoother works on r - mean(r over coupled cells).  A residual shifted by a constant on the coupled
    cells must give the same x and leave the same (mean-free) r; on a tiny periodic grid, CG on a
    residual that is ONLY a constant must not move x at all (without the projection alpha = rho/0)."""
    cfg = wi.sphere((32, 16, 16), D=8.0, centre=(8.0, 8.0, 8.0))
    out = []
    for shift in (0.0, 0.37):
        s = wo.OracleSim(cfg)
        live = s.interior("iD")[0] != 0
        assert (~live).sum() > 0                      # the body buries some cells
        r = wi.random_scalar((32, 16, 16), seed=21)
        r[~live] = 0.0
        r[live] += shift - r[live].mean()
        s.interior("r")[0][...] = r
        s.arr("x")[...] = 0.0
        s.smooth(0, 6)
        out.append((s.interior("x").copy(), s.interior("r").copy(), live))
        s.close()
    (x0, r0, live), (x1, r1, _) = out
    assert np.abs(x0).max() > 1e-3
    assert np.allclose(x1, x0, atol=1e-12) and np.allclose(r1, r0, atol=1e-12)
    assert abs(r1[0][live].mean()) < 1e-14 and np.all(r1[0][~live] == 0.0)
    s = wo.OracleSim(wi.make(ndim=2, dims=(4, 4), periodic=(1, 1), U=(0.0,) * 3))
    s.interior("r")[0, 0][...] = 0.25
    s.arr("x")[...] = 0.0
    s.smooth(0, 6)
    assert np.all(s.interior("x") == 0.0) and np.abs(s.interior("r")).max() < 1e-16
    s.close()


def test_restrict_prolong_definitions():
    s = wo.OracleSim(wi.tgv3d(8, max_levels=2))
    g = wi.rng(13)
    r = g.standard_normal((8, 8, 8))
    s.interior("r", 0)[0][...] = r
    s.restrict(0)
    rc = s.interior("r", 1)[0]
    assert np.allclose(rc, r.reshape(4, 2, 4, 2, 4, 2).sum(axis=(1, 3, 5)), atol=1e-14)
    # prolong: x_f += x_c[parent], r_f -= A e
    xc = g.standard_normal((4, 4, 4))
    s.interior("x", 1)[0][...] = xc
    s.interior("x", 0)[0][...] = 0.0
    s.prolong_increment(0)
    e = np.repeat(np.repeat(np.repeat(xc, 2, 0), 2, 1), 2, 2)
    assert np.allclose(s.interior("x", 0)[0], e, atol=1e-14)
    Ae, _ = _apply(s, 0, e)
    assert np.allclose(s.interior("r", 0)[0], r - Ae, atol=1e-13)
    s.close()


@pytest.mark.parametrize("which", ["sphere", "periodic", "circle2d"])
def test_projection_identities(which):
    """BASELINE north_star pin: the discrete divergence after projection falls to the solver
    tolerance; plus div(u_new) == final residual, idempotence, untouched boundary faces."""
    kw = dict(fixed_vcycles=0, tol=1e-10, max_vcycles=100)
    if which == "sphere":
        cfg = wi.sphere((32, 16, 16), D=8.0, centre=(8.0, 8.0, 8.0), **kw)
    elif which == "periodic":
        cfg = wi.tgv3d(16, **kw)
    else:
        cfg = wi.make(ndim=2, dims=(32, 16), periodic=(0, 1), exit_bc=1, body_kind=wi.BODY_SPHERE,
                      centre=(10.0, 8.0), R=3.0, **kw)
    s = wo.OracleSim(cfg)
    nd = cfg["ndim"]
    s.set_fields(u=wi.random_velocity(cfg["dims"][:nd], seed=31, mean=cfg["U"]))
    # cells buried in the body are decoupled (D = 0): give them a solid-consistent velocity
    # u = mu0*u (= V = 0 inside), as the BDIM blend would
    s.interior("u")[...] *= s.interior("mu0")
    s.bc()
    if cfg["exit_bc"]:
        s.arr("u0")[...] = s.arr("u")
        s.exit_bc(0.3)                              # makes the boundary flux compatible (O6)
    inner = (lambda a: a[0, 1:-1, 1:-1, 1:-1]) if nd == 3 else (lambda a: a[0, 0, 1:-1, 1:-1])
    assert abs(inner(s.divergence()).sum()) < 1e-10
    s.project(1.0, 0.25)
    s.bc()                                          # refresh periodic ghosts (O9 order: project; BC)
    dnew = inner(s.divergence())
    assert np.allclose(dnew, inner(s.arr("r")), atol=1e-12)      # identity div(u - L grad x) = z - A x
    assert np.abs(dnew).max() <= 1e-10                           # fell to the solver tolerance
    assert s.stats()["vcycles"][0] < 100
    ubefore = s.interior("u").copy()
    s.arr("p")[...] = 0.0
    s.project(1.0, 0.25)                                         # idempotent
    assert np.allclose(s.interior("u"), ubefore, atol=1e-9)
    assert np.abs(s.interior("p")).max() < 1e-8
    if not cfg["periodic"][0]:                                   # L = 0 on the inflow face
        assert np.all(s.arr("u")[0][..., 1] == cfg["U"][0])
    s.close()


# ---------------------------------------------------------------------------------------------------
# Pins for the two constants of DESIGN.md R-O and R-T that the paper does not state (P:76, P:149 name the
# solver only): the decoupling threshold |D| > 2n * 1e-6 of level_diag and the relative stop
# |rho'| < 1e-8 |rho0| of wlo_smooth.  Each test fails if the constant is changed by 100x either way.

@pytest.mark.parametrize("nd", [2, 3])
def test_level_diag_threshold_is_2n_times_1e_minus_6(nd):
    """R-O: iD = 1/D where |D| > 2n * 1e-6, else 0.  Hand-set face coefficients give cells with
    |D| = 0 (-> 0), 0.5x the threshold (-> 0), 2x the threshold (-> 1/D), 5e-6 (between the 2-D threshold
    4e-6 and the 3-D one 6e-6: coupled in 2-D, decoupled in 3-D, which pins the factor 2n), and an
    ordinary fluid cell (-> -1/2n)."""
    dims = (12, 8) if nd == 2 else (12, 8, 8)
    s = wo.OracleSim(wi.make(ndim=nd, dims=dims, periodic=(0,) * 3, U=(0.0,) * 3))
    L = s.arr("L", 0)
    thr = 2 * nd * 1e-6

    def set_cell(c0, total):
        """all 2n faces of cell (c0, 4[, 4]) get total / 2n, so that D = -total"""
        c = (4, 4, c0) if nd == 3 else (0, 4, c0)           # (c2, c1, c0)
        for i in range(nd):
            up = list(c)
            up[2 - i] += 1
            L[i][c] = total / (2 * nd)
            L[i][tuple(up)] = total / (2 * nd)
        return c

    cells = {                                                # well separated: no shared faces
        "zero": set_cell(2, 0.0), "below": set_cell(4, 0.5 * thr), "above": set_cell(6, 2.0 * thr),
        "five": set_cell(8, 5e-6),
    }
    s.poisson_update()
    iD = s.arr("iD", 0)[0]
    assert iD[cells["zero"]] == 0.0
    assert iD[cells["below"]] == 0.0                          # a threshold 100x smaller would couple it
    assert iD[cells["above"]] == pytest.approx(-1.0 / (2.0 * thr), rel=1e-12)   # 100x larger would decouple it
    if nd == 2:
        assert iD[cells["five"]] == pytest.approx(-1.0 / 5e-6, rel=1e-12)
    else:
        assert iD[cells["five"]] == 0.0
    far = (4, 6, 10) if nd == 3 else (0, 6, 10)
    assert iD[far] == pytest.approx(-1.0 / (2 * nd), rel=1e-14)
    s.close()


def _periodic_laplacian_8x8():
    T = _lap1d(8, True)
    I = sp.identity(8)
    return (sp.kron(I, T) + sp.kron(T, I)).tocsr()            # x fastest


@pytest.mark.parametrize("delta,stops_after", [(1.3e-5, 1), (1.3e-4, 2)])
def test_smoother_relative_stop_is_1e_minus_8(delta, stops_after):
    """R-T on the 8x8 periodic level of the 2-D Taylor-Green case: no body, so iD = -1/4 everywhere and the
    smoother is plain CG on the textbook Laplacian.  The residual is one eigenmode of amplitude 1 plus a
    second one of amplitude delta (eigenvalues l1 = -4 sin^2(pi/8), l2 = -2: closed forms).  One CG
    iteration removes the first mode and leaves rho'/rho0 = 5.83 delta^2 (1 + O(delta^2)):
      delta = 1.3e-5 -> 9.9e-10 < 1e-8: the call must STOP after iteration 1, leaving x off the exact solution by
                        delta |1/l1 - 1/l2| max|phi2| in the second mode (a stop at 1e-10 would go on and converge);
      delta = 1.3e-4 -> 9.9e-8 > 1e-8: the call must go ON, and iteration 2 (two eigenmodes: CG is exact after
                        two) lands on the exact solution (a stop at 1e-6 would leave it 1.6e-4 off).
    The expected iterates come from an unguarded CG written here in numpy on scipy's kron Laplacian."""
    n = 8
    s = wo.OracleSim(wi.tgv2d(n, max_levels=1))
    y, x = np.meshgrid(np.arange(n) + 0.5, np.arange(n) + 0.5, indexing="ij")
    phi1, phi2 = np.cos(2 * np.pi * x / n), np.cos(2 * np.pi * 2 * y / n)
    l1, l2 = -4 * np.sin(np.pi / n) ** 2, -4 * np.sin(2 * np.pi / n) ** 2
    assert l2 == pytest.approx(-2.0, abs=1e-15)
    r0 = phi1 + delta * phi2
    s.interior("r")[0, 0][...] = r0
    s.arr("x")[...] = 0.0
    s.smooth(0, 6)
    xo = s.interior("x")[0, 0].copy()
    # unguarded Jacobi-PCG in numpy (iD = -1/4), keeping every iterate
    A = _periodic_laplacian_8x8()
    r = r0.ravel().copy(); xk = np.zeros(n * n); iD = -0.25
    e = iD * r; rho = r @ e; rho0 = rho
    iterates, ratios = [], []
    for k in range(3):
        q = A @ e; alpha = rho / (q @ e)
        xk = xk + alpha * e; r = r - alpha * q
        iterates.append(xk.reshape(n, n).copy())
        z = iD * r; rho2 = r @ z
        ratios.append(abs(rho2 / rho0))
        e = (rho2 / rho) * e + z; rho = rho2
    assert ratios[0] == pytest.approx(delta ** 2 * (1 - l2 / l1) ** 2, rel=1e-3)
    assert (ratios[0] < 1e-8) == (stops_after == 1)
    exact = phi1 / l1 + delta * phi2 / l2
    assert np.abs(iterates[1] - exact).max() < 1e-13           # two modes: CG is exact after two iterations
    assert np.abs(xo - iterates[stops_after - 1]).max() < 1e-13
    off = np.abs(xo - exact).max()
    if stops_after == 1:
        assert off == pytest.approx(delta * abs(1 / l1 - 1 / l2) * np.abs(phi2).max(), rel=1e-3)   # stopped: second mode unsolved
        assert np.abs(xo - iterates[1]).max() > 0.5 * off                      # going on WOULD have changed x
    else:
        assert off < 1e-13
    s.close()
