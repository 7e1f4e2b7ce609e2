"""wl_energy_static (include/wl.h, wl_noalloc.cu): the entry point that allocates nothing -- its reduction scratch is a static
__device__ array of libwl -- against the existing path, wl_energy on a handle (itself checked against the oracle in
test_gpu_kernels.py).  Collected last on purpose (the suite runs with pytest -x).  Runs alone in a fresh process or after the
other tests: it depends on no state but the library's."""
import ctypes as C

import numpy as np
import pytest

import wl_inputs as wi

TOL = 2e-5          # the bound of the per-kernel parity tests (tests/test_gpu_kernels.py)


def _state(cfg, steps):
    """(padded velocity with BC-filled ghosts as a cuda tensor, wl_energy of the same state) after a few steps"""
    import torch
    from paper_2407_16032_b200 import wl
    g = wl.Sim(cfg)
    tgv = cfg["body_kind"] == 0
    if tgv:
        g.init_tgv(1)
    dt = g.cfl() if tgv else 0.25
    for k in range(steps):
        g.step(dt if k == 0 else 0.0, dt, adaptive=True)
    ref = np.array(g.energy())
    u = torch.from_numpy(g.dbg_get("u", padded=True)).cuda()
    g.close()
    return u, ref


@pytest.mark.gpu
def test_static_energy_matches_wl_energy_on_calls_in_a_row():
    import torch
    from paper_2407_16032_b200 import wl
    cases = [wi.sphere(dims=(96, 48, 40), D=16.0),        # inflow / exit / slip walls, a body: 180 blocks, a ragged last one
             wi.tgv3d(32),                                 # periodic, fewer blocks than the call before: stale partials stay behind
             wi.tgv2d(64)]                                 # 2-D
    states = [_state(c, 3) for c in cases]
    nan = float("nan")
    outs = [torch.full((2,), nan, dtype=torch.float64, device="cuda") for _ in range(5)]
    wl.energy_static(states[0][0], outs[4])                # set-up call (address look-up) outside the measured region
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # calls in a row on one stream, nothing in between: large, small, large again, 2-D
    order = [0, 1, 0, 2]
    for k, c in enumerate(order):
        wl.energy_static(states[c][0], outs[k])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0           # nothing was allocated on the device
    got = [o.cpu().numpy() for o in outs]
    for k, c in enumerate(order):
        ref = states[c][1]
        assert got[k][0] == pytest.approx(ref[0], rel=TOL), (k, c)
        assert got[k][1] == pytest.approx(ref[1], rel=TOL), (k, c)
    # fixed summation order: the same bits whatever ran before
    assert np.array_equal(got[0], got[2]) and np.array_equal(got[0], got[4])


@pytest.mark.gpu
def test_static_energy_at_the_size_limit_and_beyond():
    import torch
    from paper_2407_16032_b200 import wl
    n = (1024, 256, 256)
    assert n[0] * n[1] * n[2] == wl.STATIC_MAX_CELLS       # exactly the maximum: 65536 blocks, every scratch slot in use
    gen = torch.Generator(device="cuda").manual_seed(20240716)
    u = torch.rand((3, n[2] + 2, n[1] + 2, n[0] + 2), generator=gen, device="cuda", dtype=torch.float32) - 0.5
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    wl.energy_static(u, out)
    wl.energy_static(u, out)
    # the same sums with torch in fp64 (interior = 1 .. n of every padded axis; lower neighbours reach into the ghost layer)
    ke = 0.0
    for c in range(3):
        ke += 0.5 * float((u[c, 1:-1, 1:-1, 1:-1].double() ** 2).sum())
    ux, uy, uz = (u[c].double() for c in range(3))
    C_ = (slice(1, -1),) * 3
    zm, ym, xm = (slice(0, -2), slice(1, -1), slice(1, -1)), (slice(1, -1), slice(0, -2), slice(1, -1)), (slice(1, -1), slice(1, -1), slice(0, -2))
    wz = (uy[C_] - uy[xm]) - (ux[C_] - ux[ym])
    wx = (uz[C_] - uz[ym]) - (uy[C_] - uy[zm])
    wy = (ux[C_] - ux[zm]) - (uz[C_] - uz[xm])
    ens = 0.5 * float((wx * wx + wy * wy + wz * wz).sum())
    del ux, uy, uz, wx, wy, wz
    got = out.cpu().numpy()
    assert got[0] == pytest.approx(ke, rel=TOL) and got[1] == pytest.approx(ens, rel=TOL)
    # one plane more is beyond the maximum: rejected with a clear error before anything is launched (the buffer is never touched)
    out.fill_(-1.0)
    with pytest.raises(wl.WLError, match="WL_STATIC_MAX_CELLS") as ei:
        wl.energy_static(u, out, dims=(1024, 256, 257))
    assert "error -5" in str(ei.value)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [-1.0, -1.0]
    # bad arguments
    L = wl.load()
    d = (C.c_int * 3)(8, 8, 8)
    err = C.create_string_buffer(256)
    assert L.wl_energy_static(None, 3, d, None, C.c_void_p(out.data_ptr()), err, 256) == -1 and b"null" in err.value
    assert L.wl_energy_static(C.c_void_p(u.data_ptr()), 4, d, None, C.c_void_p(out.data_ptr()), None, 0) == -1
    d0 = (C.c_int * 3)(8, 0, 8)
    assert L.wl_energy_static(C.c_void_p(u.data_ptr()), 3, d0, None, C.c_void_p(out.data_ptr()), err, 256) == -1
