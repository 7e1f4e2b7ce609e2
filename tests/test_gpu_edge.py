"""GPU parity on the degenerate and edge configurations of the path: tolerance-mode solves (V-cycle counts must agree
with the oracle's), hierarchies of one and two levels, odd sizes (no multigrid, ragged float4 groups), the smallest
periodic box, 2-D, a thin periodic-z slab and a long thin box (both on the TMA paths).  Three whole steps from a
seeded perturbed stream, velocity against the fp64 oracle."""
import numpy as np
import pytest

import wl_inputs as wi

pytestmark = pytest.mark.gpu

CASES = {
    "tolerance_mode_sphere_64x32x32": lambda: wi.sphere((64, 32, 32), D=8.0, centre=(16.0, 16.0, 16.0), fixed_vcycles=0, tol=1e-5, max_vcycles=30),
    "one_level_32^3": lambda: wi.sphere((32, 32, 32), D=8.0, centre=(12.0, 16.0, 16.0), max_levels=1),
    "two_levels_32^3": lambda: wi.sphere((32, 32, 32), D=8.0, centre=(12.0, 16.0, 16.0), max_levels=2),
    "odd_37x20x12": lambda: wi.make(ndim=3, dims=(37, 20, 12), U=(1.0, 0, 0), nu=0.02, exit_bc=1, body_kind=wi.BODY_SPHERE,
                                    centre=(12.0, 10.0, 6.0), R=3.0),
    "periodic_8^3": lambda: wi.make(ndim=3, dims=(8, 8, 8), U=(0.0, 0, 0), nu=0.02, periodic=(1, 1, 1)),
    "2d_cylinder_128x64": lambda: wi.make(ndim=2, dims=(128, 64), U=(1.0, 0, 0), nu=0.02, exit_bc=1, body_kind=wi.BODY_SPHERE,
                                          centre=(32.0, 32.0), R=6.0),
    "slab_128x128x16_periodic_z": lambda: wi.make(ndim=3, dims=(128, 128, 16), U=(1.0, 0, 0), nu=0.02, exit_bc=1, periodic=(0, 0, 1),
                                                  body_kind=wi.BODY_SPHERE, centre=(40.0, 64.0, 8.0), R=5.0),
    # every kernel family in one small case (the one the compute-sanitizer records of profiles/ run): level 0 takes the TMA-fed
    # conv_diff and the one-sweep smoother, level 1 (131 K cells) the cooperative kernel, levels 2-4 the on-chip cluster kernel
    "all_kernels_256x64x64_heaving": lambda: wi.heaving_sphere((256, 64, 64), D=16.0, centre=(64.0, 32.0, 32.0)),
    "long_256x16x16": lambda: wi.make(ndim=3, dims=(256, 16, 16), U=(1.0, 0, 0), nu=0.02, exit_bc=1, body_kind=wi.BODY_SPHERE,
                                      centre=(40.0, 8.0, 8.0), R=3.0),
}


@pytest.mark.parametrize("name", list(CASES))
def test_three_steps_vs_oracle(name):
    from oracle import wl_oracle as wo
    from paper_2407_16032_b200 import wl
    cfg = CASES[name]()
    o, g = wo.OracleSim(cfg), wl.Sim(cfg)
    nd = cfg["ndim"]
    dims = cfg["dims"][:nd]
    u0 = wi.random_velocity(dims, seed=5) * 0.3 + np.array(cfg["U"][:nd]).reshape((nd,) + (1,) * nd)
    o.set_fields(u=u0)
    g.set_fields(u=np.ascontiguousarray(u0, dtype=np.float32))
    moving = cfg["motion"] != wi.MOTION_STATIC
    for k in range(3):
        if moving:
            o.measure(0.25 * (k + 1)); g.measure(0.25 * (k + 1))
        o.mom_step(0.25)
        g.mom_step(0.25)
        assert g.stats()["vcycles"] == list(o.stats()["vcycles"])
    if moving:
        Fo, Fg = o.pressure_force(0.75), g.pressure_force(0.75)
        assert np.abs(Fg - Fo).max() <= 1e-3 * np.abs(Fo).max()
    u, _p = g.fields()
    uo = o.interior("u")
    uo = uo[:, 0] if nd == 2 else uo
    assert np.abs(u - uo).max() <= 1e-4 * np.abs(uo).max()
    assert g.stats()["nan_flag"] == 0
    o.close(); g.close()
