"""GPU parity of the alternative kernel paths of the projection: the shared-memory PCG pass A
(`k_pcg_A_fast`) against the register-marching one, the persistent coarse-level kernels (`k_coarse`, cooperative;
`k_tiny`, one thread-block cluster) against stand-alone launches, a fused chain of coarse passes against the same
passes launched one by one -- each against the fp64 oracle, and against one another.  The paths are chosen by the `tune` entry of the config
(wl_tuning in include/wl.h), copied into the handle when a simulation is created."""

import numpy as np
import pytest

import wl_inputs as wi
from test_gpu_kernels import CASES, O, TOL, _cfg, _ids, _load_state, _sims, diag, relerr

pytestmark = pytest.mark.gpu

SWITCHES = [
    {},                                     # default: fast pass A, k_coarse for levels <= 1 M cells, k_tiny below
    {"no_fused": 1},                        # two-pass PCG iterations (wl_pcgfast.cu pass A + k_pcg_B) instead of the one-sweep form
    {"no_fast_a": 1},                       # register-marching pass A everywhere
    {"no_block_levels": 1},                 # small levels inside the cooperative kernel
    {"pk_max_cells": -1},                   # every level by stand-alone kernels
    {"no_bulk": 1},                         # pass A copies its planes with per-thread cp.async instead of TMA boxes
    {"no_tma_cd": 1},                       # conv_diff from the register-staged ring (k_cd_tile2) instead of the TMA-fed one
    {"pk_fail": 1},                         # the device refuses the cluster and the cooperative launch: fallback to stand-alone passes
]


def _tuned(cfg, sw):
    return dict(cfg, tune=dict(sw))


# the last two take the TMA path of pass A (rows of whole 128-cell tiles, no wrap in x and y)
WIDE = [c for c in CASES if len(c[0]) == 3 and c[0][0] >= 136] + [((64, 64, 64), (0, 1, 0), 1, "sphere", False),
                                                                   ((128, 40, 24), (0, 0, 0), 1, "sphere", False),
                                                                   ((256, 24, 20), (0, 0, 1), 1, "torus", False)]


@pytest.mark.parametrize("case", WIDE, ids=_ids)
def test_every_path_matches_the_oracle_and_the_others(case):
    """Three full steps (fixed two V-cycles) through each path: velocity vs the oracle <= 1e-4, and the paths
    agree with one another to round-off amplified by three steps."""
    from oracle import wl_oracle as wo
    from paper_2407_16032_b200 import wl
    cfg = _cfg(case)
    o = wo.OracleSim(cfg)
    u0 = wi.random_velocity(case[0], seed=wi.SEED + 3)
    o.set_fields(u=u0)
    dt = 0.25
    for _ in range(3):
        o.mom_step(dt)
    uo = O(o, "u")
    outs = []
    for sw in SWITCHES:
        g = wl.Sim(_tuned(cfg, sw))
        g.set_fields(u=np.ascontiguousarray(u0, dtype=np.float32))
        for _ in range(3):
            g.mom_step(dt)
        u, _p = g.fields()
        assert g.stats()["nan_flag"] == 0
        assert relerr(u, uo) <= 1e-4, sw
        outs.append(u.astype(np.float64))
        g.close()
    for u in outs[1:]:
        assert np.abs(u - outs[0]).max() <= 2e-5 * np.abs(uo).max()
    o.close()


@pytest.mark.parametrize("case", [CASES[0], CASES[2], CASES[8], CASES[9]], ids=_ids)
def test_fused_coarse_chain_equals_single_passes(case):
    """The V-cycle below level 0 as ONE chain (wl_dbg_coarse_prog) and as one launch per pass give the oracle's
    x and r on every level; after each smooth the stored sum of r over the coupled cells is reset (R-T2)."""
    cfg = _cfg(case)
    dims = case[0]
    res = []
    for fused in (True, False):
        o, g = _sims(cfg)
        _load_state(o, g, dims)
        o.arr("u0")[...] = o.arr("u"); g.dbg_save_u0()
        o.conv_diff("u0"); o.bdim(0.3, 0); g.dbg_conv_diff_bdim(0.3, 0)
        o.bc(); g.dbg_bc()
        if case[2]:
            o.exit_bc(0.3); g.dbg_exit_bc(0.3)
        x0 = np.zeros(dims[::-1])
        o.interior("x")[0][...] = x0; g.dbg_set("x", x0[None].astype(np.float32))
        o.arr("sig")[...] = o.divergence(); o.residual(); g.dbg_residual()
        n = o.nlevels
        ops = []
        for l in range(n - 1):
            o.restrict(l); o.arr("x", l + 1)[...] = 0.0
            ops.append((0, l, 0))
        for l in range(n - 1, 0, -1):
            o.smooth(l, 6); ops.append((1, l, 6))
            o.prolong_increment(l - 1); ops.append((2, l - 1, 0))
        if fused:
            g.dbg_coarse_prog(ops)
        else:
            for op in ops:
                g.dbg_coarse_prog([op])
        r0 = np.abs(O(o, "r", 0)).max()
        lev = []
        for l in range(n):
            xg, rg = g.dbg_get("x", l), g.dbg_get("r", l)
            assert relerr(xg, O(o, "x", l)) <= 1e-4
            assert np.abs(rg - O(o, "r", l)).max() <= 1e-4 * max(r0, np.abs(O(o, "r", l)).max())
            lev.append((xg, rg))
        for l in range(1, n):
            sc = g.dbg_pcg_scalars(l)
            assert sc["rsum"] == 0.0                                   # reset by the smoother
            assert sc["nlive"] == float((O(o, "iD", l)[0] != 0).sum())
        res.append(lev)
        o.close(); g.close()
    for (xa, ra), (xb, rb) in zip(*res):
        assert np.array_equal(xa, xb) and np.array_equal(ra, rb)       # same kernels, same order: bit-identical


@pytest.mark.parametrize("kernel", ["tile2", "tile3"])
@pytest.mark.parametrize("case", [c for c in WIDE if not c[1][0] and not c[1][1]] + [CASES[1], CASES[4]], ids=_ids)
def test_conv_diff_kernels_agree(case, kernel):
    """conv_diff + BDIM + Heun through each of the two tile kernels (k_cd_tile2, the TMA-fed k_cd_tile3 where x and
    y do not wrap): predictor and corrector against the oracle at the per-kernel tolerance."""
    from paper_2407_16032_b200 import wl
    cfg = _cfg(case)
    for corrector in (0, 1):
        o, _g = _sims(cfg)
        _g.close()
        g = wl.Sim(_tuned(cfg, {"no_tma_cd": 1} if kernel == "tile2" else {}))
        _load_state(o, g, case[0], seed=wi.SEED, p_too=False)
        o.arr("u0")[...] = o.arr("u"); g.dbg_save_u0()
        if corrector:
            _load_state(o, g, case[0], seed=wi.SEED + 11, p_too=False)
            o.conv_diff("u")
        else:
            o.conv_diff("u0")
        o.bdim(0.31, corrector); g.dbg_conv_diff_bdim(0.31, corrector)
        assert relerr(g.dbg_get("u"), O(o, "u")) <= TOL
        o.close(); g.close()


def test_smoother_removes_residual_mean_on_the_gpu():
    """R-T2 on the device: a residual shifted by a constant on the coupled cells gives the same x (oracle pin
    test_smoother_removes_the_incompatible_part_of_the_residual, here for libwl on every level)."""
    cfg = _cfg(CASES[8])
    o, g = _sims(cfg)
    for l in range(o.nlevels):
        ld = g.level_dims(l)
        live = O(o, "iD", l)[0] != 0
        out = []
        for shift in (0.0, 0.05):
            r = wi.random_scalar(ld, seed=500 + l)
            r = r * np.minimum(1.0, np.abs(diag(O(o, "iD", l)[0])))
            r[~live] = 0.0
            r[live] += shift - r[live].mean()
            g.dbg_set("r", r[None].astype(np.float32), l)
            g.dbg_set("x", np.zeros_like(r)[None].astype(np.float32), l)
            g.dbg_smooth(l, 3)
            out.append((g.dbg_get("x", l).astype(np.float64), g.dbg_get("r", l).astype(np.float64)))
        (xa, ra), (xb, rb) = out
        # the shifted residual is rounded to fp32 before the smoother sees it: 3 CG iterations amplify that round-off
        assert np.abs(xb - xa).max() <= 1e-4 * max(np.abs(xa).max(), 1e-30)
        assert abs(rb[0][live].mean()) <= 1e-6
    o.close(); g.close()


# levels the one-sweep smoother (wl_pcgfused.cu) takes: 3-D, at least 68 cells along x; with
# pk_max_cells = -1 level 1 of the second case (128 x 16 x 12) is a stand-alone level too and takes it as well
FUSED = [((128, 40, 24), (0, 0, 0), 1, "sphere", False), ((256, 32, 24), (0, 0, 1), 1, "torus", False),
         ((160, 44, 24), (0, 0, 0), 1, "sphere", False),          # rows of 1.25 tiles, 5.5 tiles along y
         # levels that wrap in x and / or y: the arrays read with halos carry periodic ghost cells (a TMA box cannot wrap)
         ((136, 40, 24), (1, 1, 1), 0, "torus", False),           # ragged row end on a periodic x
         ((256, 32, 24), (1, 1, 0), 0, "sphere", False),          # levels 0 and 1
         ((160, 44, 24), (0, 1, 0), 1, "sphere", False)]          # ragged last row of tiles on a periodic y


def _fused_levels(case):
    return (0, 1) if case[0][0] == 256 else (0,)


def _smoother_inputs(o, g, l):
    ld = g.level_dims(l)
    r0 = wi.random_scalar(ld, seed=700 + l)
    r0 -= r0.mean()
    r0 = r0 * np.minimum(1.0, np.abs(diag(O(o, "iD", l)[0])))
    g.dbg_set("L", O(o, "L", l), l)
    g.dbg_set("iD", O(o, "iD", l), l)
    return r0


def _run_smoother(o, g, l, r0, iters):
    o.interior("r", l)[0][...] = r0
    o.arr("x", l)[...] = 0.0
    g.dbg_set("r", r0[None].astype(np.float32), l)
    g.dbg_set("x", np.zeros_like(r0)[None].astype(np.float32), l)
    o.smooth(l, iters)
    g.dbg_smooth(l, iters)
    return g.dbg_get("x", l), g.dbg_get("r", l)


@pytest.mark.parametrize("iters", [1, 2, 3, 6])
@pytest.mark.parametrize("case", FUSED, ids=_ids)
def test_one_sweep_smoother_matches_the_oracle_and_the_two_pass_form(case, iters):
    """The recurrence form of the PCG iteration (one sweep per iteration, r and q ping-pong: odd and even numbers of
    swaps) against the oracle and against the two-pass kernels, on levels 0 and 1."""
    from paper_2407_16032_b200 import wl
    cfg = _cfg(case)
    outs = []
    for sw in ({"pk_max_cells": -1}, {"pk_max_cells": -1, "no_fused": 1}):
        o, g0 = _sims(cfg)
        g0.close()
        g = wl.Sim(_tuned(cfg, sw))
        res = []
        for l in _fused_levels(case):
            r0 = _smoother_inputs(o, g, l)
            g.prof_enable(True)
            xg, rg = _run_smoother(o, g, l, r0, iters)
            prof = g.prof_read()
            g.prof_enable(False)
            # no silent change of path: the one-sweep form is iters - 1 fused sweeps, the two-pass form none
            nfused = sum(n for k, (_ms, n) in prof.items() if k.startswith("pcg_fused"))
            assert nfused == (0 if "no_fused" in sw else iters - 1), (sw, l, prof)
            tol = TOL if iters == 1 else 1e-4
            assert relerr(xg, O(o, "x", l)) <= tol, (sw, l)
            assert np.abs(rg - O(o, "r", l)).max() <= tol * np.abs(r0).max(), (sw, l)
            res.append((xg.astype(np.float64), rg.astype(np.float64), np.abs(r0).max()))
        outs.append(res)
        o.close(); g.close()
    for (xa, ra, s), (xb, rb, _s) in zip(*outs):
        assert np.abs(xa - xb).max() <= 1e-4 * np.abs(xb).max()
        assert np.abs(ra - rb).max() <= 1e-4 * s


@pytest.mark.parametrize("case", FUSED, ids=_ids)
def test_one_sweep_smoother_stops_like_the_oracle(case):
    """R-T guards in the one-sweep form.  A zero residual changes nothing.  A residual scaled so that |rho| falls below
    tau = 1e-30 after the first iteration stops the oracle there; the device evaluates the criterion on the recurrence
    value of rho', applies the update still owed in the next sweep and carries r across the remaining ones: x and r
    as the oracle's."""
    from paper_2407_16032_b200 import wl
    cfg = _cfg(case)
    o, g0 = _sims(cfg)
    g0.close()
    g = wl.Sim(_tuned(cfg, {"pk_max_cells": -1}))
    for l in _fused_levels(case):
        r0 = _smoother_inputs(o, g, l)
        iD = O(o, "iD", l)[0]
        # zero residual
        x1 = wi.random_scalar(g.level_dims(l), seed=800 + l).astype(np.float32)
        g.dbg_set("r", np.zeros_like(r0)[None].astype(np.float32), l)
        g.dbg_set("x", x1[None], l)
        g.dbg_smooth(l, 6)
        assert np.array_equal(g.dbg_get("x", l)[0], x1) and not g.dbg_get("r", l).any()
        assert g.dbg_pcg_scalars(l)["live"] == 0.0
        # a checkerboard is (away from boundaries and the body) an eigenvector of iD A: one iteration takes |rho| = |r . iD r|
        # down by ~1e3.  |rho_k| of the unscaled problem after k iterations, from the oracle's residuals:
        shp = o.interior("r", l)[0].shape
        k3, j3, i3 = np.indices(shp)
        rc = (1.0 - 2.0 * ((i3 + j3 + k3) & 1)) * np.minimum(1.0, np.abs(diag(iD))) + 0.02 * r0
        rc -= rc.mean()
        rho = []
        for k in range(3):
            o.interior("r", l)[0][...] = rc
            o.arr("x", l)[...] = 0.0
            if k:
                o.smooth(l, k)
            rk = O(o, "r", l)[0]
            rho.append(abs(float((rk * iD * rk).sum())))
        assert rho[1] <= rho[0] / 64.0
        scale = np.sqrt(1e-30 * 8.0 / rho[0])                 # rho_0 = 8 tau, rho_1 <= tau / 8: the smoother stops after one iteration
        for iters in (1, 2, 3, 6):                            # the update still owed is applied by the last sweep / a fused sweep
            xg, rg = _run_smoother(o, g, l, rc * scale, iters)
            xo, ro = O(o, "x", l).copy(), O(o, "r", l).copy()
            o.interior("r", l)[0][...] = rc * scale
            o.arr("x", l)[...] = 0.0
            o.smooth(l, 1)
            # the oracle did stop after the first iteration (its OpenMP sums may differ in the last bit from run to run)
            assert np.allclose(O(o, "x", l), xo, rtol=1e-10, atol=0.0)
            assert g.dbg_pcg_scalars(l)["live"] == 0.0
            assert relerr(xg, xo) <= 1e-4, (l, iters)
            assert np.abs(rg - ro).max() <= 1e-4 * np.abs(rc * scale).max(), (l, iters)
    o.close(); g.close()


@pytest.mark.parametrize("case", [c for c in CASES if c[4]] + [((160, 48, 40), (0, 0, 1), 1, "sphere", True)], ids=_ids)
def test_poisson_update_inside_the_body_box_equals_a_full_update(case):
    """After the first measure!, mu0, L, 1/D, the tile modes and the count of coupled cells are recomputed only in the box the
    moving body can reach: after several measures the arrays of every level are bit-identical to those of a fresh handle
    measured once at the last time (a full update), and the counts equal the oracle's."""
    from paper_2407_16032_b200 import wl
    cfg = _cfg(case)
    o, g = _sims(cfg)
    for t in (1.7, 4.1, 9.6, 13.2):
        g.measure(t)
    o.measure(13.2)
    f = wl.Sim(cfg)
    f.measure(13.2)
    for l in range(o.nlevels):
        for name in ("L", "iD"):
            assert np.array_equal(g.dbg_get(name, l, padded=True), f.dbg_get(name, l, padded=True)), (name, l)
        assert g.dbg_pcg_scalars(l)["nlive"] == f.dbg_pcg_scalars(l)["nlive"] == float((O(o, "iD", l)[0] != 0).sum())
    o.close(); g.close(); f.close()


@pytest.mark.parametrize("amp", [0.0, 1e-19])
def test_solve_whose_smoother_has_nothing_to_do(amp):
    """A uniform stream without a body is divergence-free: the residual of both projections is zero (amp = 0) or so small that
    |rho| < tau stops the smoother in its first sweep (amp = 1e-19), on every level.  The updates that the one-sweep smoother
    leaves to restrict(0), prolong(0) and apply_gradient are then NOT owed: the stream must come out untouched
    (amp = 0: bit for bit) and as the oracle's."""
    from oracle import wl_oracle as wo
    from paper_2407_16032_b200 import wl
    cfg = wi.make(ndim=3, dims=(136, 40, 24), U=(1.0, 0.0, 0.0), nu=0.02, exit_bc=1)
    o, g = wo.OracleSim(cfg), wl.Sim(cfg)
    u0 = np.zeros((3, 24, 40, 136)); u0[0] = 1.0
    if amp:
        u0 += amp * wi.random_velocity((136, 40, 24), seed=3)
    o.set_fields(u=u0)
    g.set_fields(u=np.ascontiguousarray(u0, dtype=np.float32))
    for k in range(2):
        o.mom_step(0.25); g.mom_step(0.25)
    u, p = g.fields()
    assert g.stats()["nan_flag"] == 0 and np.isfinite(u).all() and np.isfinite(p).all()
    assert np.abs(u - o.interior("u")).max() <= 1e-6
    if amp == 0.0:
        assert np.array_equal(u[0], np.ones_like(u[0])) and not u[1:].any() and not p.any()
    o.close(); g.close()
