"""CPU-side checks of the boundary: libwl.so builds with nvcc (cross-compiled, no GPU needed),
loads, and exports every symbol include/wl.h declares; pure host functions behave.  No compute
call is made here."""
import ctypes as C
import re
from pathlib import Path

import pytest

import wl_inputs as wi

ROOT = Path(__file__).resolve().parent.parent


def _declared():
    text = (ROOT / "include" / "wl.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(wl_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2407_16032_b200 import wl
    L = wl.load()
    names = _declared()
    assert len(names) >= 25
    for n in names:
        assert hasattr(L, n), f"libwl.so does not export {n}"
    assert sorted(wl.EXPORTS) == names
    assert L.wl_abi_version() == 2


def test_config_struct_layout_matches_header():
    """The ctypes mirror must have the C layout: all members are 4-byte scalars, no padding."""
    from paper_2407_16032_b200 import wl
    assert C.sizeof(wl.Body) == 4 * (1 + 3 + 2 + 1 + 1 + 9 + 1 + 5 + 1)
    assert C.sizeof(wl.MG) == 4 * 5
    assert C.sizeof(wl.Tuning) == 4 * 6 + 8 + 8              # six ints, one long long (8-aligned), two ints
    head = 4 * (1 + 3 + 1 + 3 + 1 + 3 + 1 + 1 + 4) + C.sizeof(wl.Body) + C.sizeof(wl.MG)
    assert wl.Config.tune.offset == (head + 7) // 8 * 8
    tail = 4 + 3 * C.sizeof(wl.Body) + 4 * 3 + 4 * 3          # nextra, extra[3], extra_op[3]; precision, tangent_param, tangent_index
    assert wl.Config.nextra.offset == wl.Config.tune.offset + C.sizeof(wl.Tuning)
    assert C.sizeof(wl.Config) == (wl.Config.nextra.offset + tail + 7) // 8 * 8


def test_workspace_bytes_is_pure_and_sane():
    from paper_2407_16032_b200 import wl
    for k in range(5):
        cfg = wi.baseline_config(k)
        n = wl.workspace_bytes(cfg)
        cells = 1
        for d in cfg["dims"][: cfg["ndim"]]:
            cells *= d
        assert n > 0 and n == wl.workspace_bytes(cfg)
        if k >= 3:
            # SURVEY 8(a) P0 / PAPER.md:165: about 32 floats = 128 B per cell
            assert 100 <= n / cells <= 135
    assert wl.workspace_bytes(wi.make(ndim=3, dims=(3, 8, 8))) == 0
    assert wl.workspace_bytes(wi.make(ndim=3, dims=(8, 8, 8), eps=0.0)) == 0
    bad = wi.make(ndim=2, dims=(8, 8), body_kind=wi.BODY_TORUS)
    assert wl.workspace_bytes(bad) == 0


def test_create_rejects_bad_arguments_without_gpu():
    """Argument validation happens before any CUDA call."""
    from paper_2407_16032_b200 import wl
    L = wl.load()
    c = wl.make_config(wi.make(ndim=3, dims=(8, 8, 8)))
    h = C.c_void_p()
    assert L.wl_sim_create(C.byref(c), None, 0, None, C.byref(h)) == wl.WL_ENOMEM
    assert L.wl_sim_create(C.byref(c), C.c_void_p(1024 + 8), 1 << 40, None, C.byref(h)) == wl.WL_ENOMEM   # misaligned
    c.ndim = 5
    assert L.wl_sim_create(C.byref(c), None, 0, None, C.byref(h)) == wl.WL_EINVAL
    assert L.wl_mom_step(None, 0.1) == wl.WL_EINVAL


def test_library_reads_no_environment_variable():
    """include/wl.h promises 'no global state': the implementation switches travel in wl_config.tune."""
    for path in (ROOT / "paper_2407_16032_b200" / "csrc").iterdir():
        assert "getenv" not in path.read_text(), path


def test_product_never_imports_the_oracle():
    for path in (ROOT / "paper_2407_16032_b200").rglob("*"):
        if path.suffix in (".py", ".cu", ".cuh", ".h"):
            text = path.read_text()
            assert "wl_oracle" not in text and "wlo_" not in text, path
            assert not re.search(r"(import|from)\s+oracle", text), path


def test_sim_fails_loudly_without_cuda():
    import torch
    from paper_2407_16032_b200 import wl
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        wl.Sim(wi.baseline_config(0))
