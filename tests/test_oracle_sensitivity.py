"""How far the METHOD itself amplifies round-off over the north_star's ten-step horizon: the fp64 oracle against a copy
of itself whose velocity is perturbed by 1e-7 (Gaussian, seeded) after the first step, BASELINE configs[3] (the bench
workload C4: torus, Re = 1000) at 1/2 linear scale, two fixed V-cycles.  CPU only; about 40 s on 8 cores.

What it records (tests/test_gpu_fullsize.py holds the CUDA path to the matching statement at
full size): the perturbation grows by more than two orders of magnitude on a handful of faces hugging the torus
surface, where a flux-limiter branch of the QUICK scheme flips, while the field as a whole stays at the
size of the perturbation.  So no fp32 implementation can hold 1e-4 in L-infinity over ten steps on those faces, and
the ten-step bound is stated on the faces away from the body plus the 99.9th percentile."""
import numpy as np

import wl_inputs as wi
from oracle import wl_oracle as wo


def _ten_steps(cfg, perturb=None):
    o = wo.OracleSim(cfg)
    dt, dts = cfg["dt0"], []
    for k in range(10):
        o.mom_step(dt)
        dts.append(dt)
        if k == 0 and perturb:
            ui = o.interior("u")
            ui[...] += perturb * wi.rng(99).standard_normal(ui.shape)
            o.bc()
        dt = o.cfl()
    u = o.interior("u").copy()
    o.close()
    return u


def test_c4_half_scale_amplifies_1e_minus_7_locally_not_globally():
    cfg = wi.baseline_config(3, scale=2)                  # 256 x 128 x 128, torus R 16, r 4 at (64, 64, 64)
    assert cfg["fixed_vcycles"] == 2
    a = _ten_steps(cfg)
    b = _ten_steps(cfg, perturb=1e-7)
    sc = np.abs(a).max()
    d = np.abs(a - b) / sc
    linf, p999 = d.max(), np.percentile(d, 99.9)
    print(f"oracle vs perturbed oracle, C4 at 1/2 scale, 10 steps: rel Linf {linf:.3e}, 99.9th percentile {p999:.2e}, "
          f"share of faces above 1e-5: {(d > 1e-5).mean():.2e}")
    # amplified by more than 300x somewhere (measured 2.1e-4: a factor 2000) ...
    assert linf >= 3e-5
    # ... but not as a field: 99.9 % of the faces stay within 10x the perturbation (measured 1.3e-7)
    assert p999 <= 1e-6
    assert (d > 1e-5).mean() <= 1e-4                      # measured 1.3e-5 of the faces
    # ... and the eight largest differences sit within three cells of the torus surface (measured 1.0 .. 1.7 cells)
    nx, ny, nz = cfg["dims"]
    cx, cy, cz = cfg["centre"]
    for flat in np.argsort(d.ravel())[-8:]:
        comp, z, y, x = np.unravel_index(flat, d.shape)
        pos = [x + 0.5 - cx, y + 0.5 - cy, z + 0.5 - cz]
        pos[comp] -= 0.5                                  # the face sits half a cell below the centre
        sdf = np.sqrt((np.sqrt(pos[1] ** 2 + pos[2] ** 2) - cfg["R"]) ** 2 + pos[0] ** 2) - cfg["r"]
        assert abs(sdf) <= 3.0, (comp, z, y, x, sdf, d[comp, z, y, x])
