"""Thin Python binding of libwl (include/wl.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of libwl.so; PyTorch is used for device memory
(the workspace and user buffers) and the stream.  There is no CPU fallback: importing works
without a GPU (so the ABI can be checked), but creating a simulation without the built library
or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import math
from pathlib import Path

import numpy as np

from . import build as _build

BODY_NONE, BODY_SPHERE, BODY_TORUS, BODY_CYLINDER, BODY_PLANE = 0, 1, 2, 3, 4
MOTION_STATIC, MOTION_SIN = 0, 1
WL_OK, WL_EINVAL, WL_ENOMEM, WL_ECUDA, WL_ENOCONV = 0, -1, -2, -3, -4
SEEDS = {"nu": 1, "U": 2, "R": 3, "spin": 4, "amp": 5, "centre": 6}       # WL_SEED_*: the parameter a tangent is taken with respect to

EXPORTS = [
    "wl_workspace_bytes", "wl_sim_create", "wl_sim_destroy", "wl_set_fields", "wl_init_tgv", "wl_measure",
    "wl_mom_step", "wl_cfl", "wl_pressure_force", "wl_energy", "wl_get_fields", "wl_step",
    "wl_get_fields_f64", "wl_set_fields_f64", "wl_pressure_force_f64", "wl_energy_f64", "wl_dbg_get_f64",
    "wl_dbg_conv_diff_bdim", "wl_dbg_save_u0", "wl_dbg_bc", "wl_dbg_exit_bc", "wl_dbg_project",
    "wl_dbg_residual", "wl_dbg_apply_gradient", "wl_dbg_restrict", "wl_dbg_prolong", "wl_dbg_smooth", "wl_dbg_vcycle",
    "wl_dbg_coarse_prog", "wl_dbg_pcg_scalars",
    "wl_dbg_get", "wl_dbg_set", "wl_dbg_get_padded", "wl_level_dims", "wl_last_error", "wl_stats", "wl_abi_version",
    "wl_prof_enable", "wl_prof_read", "wl_energy_static",
]


class Body(C.Structure):
    _fields_ = [("kind", C.c_int), ("centre", C.c_float * 3), ("R", C.c_float), ("r", C.c_float),
                ("axis", C.c_int), ("motion", C.c_int),
                ("amp", C.c_float * 3), ("freq", C.c_float * 3), ("phase", C.c_float * 3),
                ("shell", C.c_float), ("scale_amp", C.c_float * 3), ("scale_freq", C.c_float), ("scale_phase", C.c_float),
                ("spin", C.c_float)]


class MG(C.Structure):
    _fields_ = [("max_levels", C.c_int), ("smooth_iters", C.c_int), ("max_vcycles", C.c_int),
                ("fixed_vcycles", C.c_int), ("tol", C.c_float)]


class Tuning(C.Structure):
    _fields_ = [("no_fused", C.c_int), ("no_fast_a", C.c_int), ("no_bulk", C.c_int), ("no_block_levels", C.c_int),
                ("no_tma_cd", C.c_int), ("zc", C.c_int), ("pk_max_cells", C.c_longlong), ("pk_blocks_per_sm", C.c_int),
                ("pk_fail", C.c_int)]


class Config(C.Structure):
    _fields_ = [("ndim", C.c_int), ("dims", C.c_int * 3), ("L", C.c_float), ("U", C.c_float * 3),
                ("nu", C.c_float), ("periodic", C.c_int * 3), ("exit_bc", C.c_int), ("eps", C.c_float),
                ("dt0", C.c_float), ("dt_max", C.c_float), ("cfl_c", C.c_float), ("cfl_cnu", C.c_float),
                ("body", Body), ("mg", MG), ("tune", Tuning),
                ("nextra", C.c_int), ("extra", Body * 3), ("extra_op", C.c_int * 3),
                ("precision", C.c_int), ("tangent_param", C.c_int), ("tangent_index", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("vcycles", C.c_int * 2), ("res", C.c_double * 2), ("nlevels", C.c_int),
                ("kernel_launches", C.c_int), ("nan_flag", C.c_int), ("noconv", C.c_int)]


_lib = None


def lib_path() -> Path:
    return _build.LIB


def load(build_if_missing: bool = True):
    """Load libwl.so (building it with nvcc when missing).  Fails loudly; never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build() if build_if_missing else _build.LIB
    if not Path(path).exists():
        raise RuntimeError(f"libwl.so not built at {path}: run python -m paper_2407_16032_b200.build")
    L = C.CDLL(str(path))
    vp, fp, ip = C.c_void_p, C.POINTER(C.c_float), C.c_int
    L.wl_workspace_bytes.restype = C.c_size_t
    L.wl_workspace_bytes.argtypes = [C.POINTER(Config)]
    L.wl_sim_create.argtypes = [C.POINTER(Config), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.wl_sim_destroy.argtypes = [vp]
    L.wl_set_fields.argtypes = [vp, vp, vp, ip]
    L.wl_init_tgv.argtypes = [vp, ip]
    L.wl_measure.argtypes = [vp, C.c_double]
    L.wl_mom_step.argtypes = [vp, C.c_float]
    L.wl_step.argtypes = [vp, C.c_double, C.c_float, ip]
    L.wl_cfl.argtypes = [vp, fp]
    L.wl_pressure_force.argtypes = [vp, C.c_double, fp]
    L.wl_energy.argtypes = [vp, C.POINTER(C.c_double)]
    dp = C.POINTER(C.c_double)
    L.wl_get_fields_f64.argtypes = [vp, vp, vp, ip, ip]
    L.wl_set_fields_f64.argtypes = [vp, vp, vp, ip]
    L.wl_pressure_force_f64.argtypes = [vp, C.c_double, dp, dp]
    L.wl_energy_f64.argtypes = [vp, dp, dp]
    L.wl_dbg_get_f64.argtypes = [vp, C.c_char_p, ip, ip, vp, C.c_size_t]
    L.wl_get_fields.argtypes = [vp, vp, vp, vp, ip]
    L.wl_dbg_conv_diff_bdim.argtypes = [vp, C.c_float, ip]
    L.wl_dbg_save_u0.argtypes = [vp]
    L.wl_dbg_bc.argtypes = [vp]
    L.wl_dbg_exit_bc.argtypes = [vp, C.c_float]
    L.wl_dbg_project.argtypes = [vp, C.c_float, C.c_float]
    L.wl_dbg_residual.argtypes = [vp]
    L.wl_dbg_apply_gradient.argtypes = [vp]
    for name in ("wl_dbg_restrict", "wl_dbg_prolong", "wl_dbg_vcycle"):
        getattr(L, name).argtypes = [vp, ip]
    L.wl_dbg_smooth.argtypes = [vp, ip, ip]
    L.wl_dbg_coarse_prog.argtypes = [vp, ip, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.wl_dbg_pcg_scalars.argtypes = [vp, ip, C.POINTER(C.c_double)]
    L.wl_dbg_get.argtypes = [vp, C.c_char_p, ip, vp, C.c_size_t]
    L.wl_dbg_set.argtypes = [vp, C.c_char_p, ip, vp, C.c_size_t]
    L.wl_dbg_get_padded.argtypes = [vp, C.c_char_p, ip, vp, C.c_size_t]
    L.wl_level_dims.argtypes = [vp, ip, C.POINTER(C.c_int)]
    L.wl_last_error.restype = C.c_char_p
    L.wl_last_error.argtypes = [vp]
    L.wl_stats.argtypes = [vp, C.POINTER(Stats)]
    L.wl_abi_version.restype = ip
    L.wl_prof_enable.argtypes = [vp, ip]
    L.wl_prof_read.argtypes = [vp, ip, C.c_char_p, C.c_size_t, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    L.wl_energy_static.restype = ip
    L.wl_energy_static.argtypes = [vp, ip, C.POINTER(C.c_int), vp, vp, C.c_char_p, C.c_size_t]
    _lib = L
    return L


def _fill_body(b: Body, d: dict) -> None:
    """one primitive (wl_body) from a plain dict; missing keys take the defaults of wl_inputs.CONFIG_DEFAULTS"""
    b.kind = int(d["kind"])
    ctr = d.get("centre", (0.0, 0.0, 0.0))
    for k in range(3):
        b.centre[k] = float(ctr[k]) if k < len(ctr) else 0.0
        b.scale_amp[k] = float((d.get("scale_amp") or (0.0, 0.0, 0.0))[k])
    b.R, b.r, b.axis, b.motion = float(d.get("R", 0.0)), float(d.get("r", 0.0)), int(d.get("axis", 0)), int(d.get("motion", MOTION_STATIC))
    # sinusoidal translation: three-vectors amp3 / freq3 / phase3, or the scalars amp / freq / phase along heave_dir
    if d.get("amp3") is not None:
        for k in range(3):
            b.amp[k], b.freq[k], b.phase[k] = float(d["amp3"][k]), float(d["freq3"][k]), float(d["phase3"][k])
    else:
        k = int(d.get("heave_dir", 1))
        b.amp[k], b.freq[k], b.phase[k] = float(d.get("amp", 0.0)), float(d.get("freq", 0.0)), float(d.get("phase", 0.0))
    b.shell, b.scale_freq, b.scale_phase = float(d.get("shell", 0.0)), float(d.get("scale_freq", 0.0)), float(d.get("scale_phase", 0.0))
    b.spin = float(d.get("spin", 0.0))


def make_config(cfg: dict) -> Config:
    """Plain dict (wl_inputs.make) -> wl_config."""
    c = Config()
    nd = int(cfg["ndim"])
    c.ndim = nd
    for d in range(3):
        c.dims[d] = int(cfg["dims"][d]) if d < nd else 1
        c.U[d] = float(cfg["U"][d]) if d < len(cfg["U"]) else 0.0
        c.periodic[d] = int(cfg["periodic"][d]) if d < nd else 0
        c.body.centre[d] = float(cfg["centre"][d]) if d < len(cfg["centre"]) else 0.0
    for k in ("L", "nu", "eps", "dt0", "dt_max", "cfl_c", "cfl_cnu"):
        setattr(c, k, float(cfg[k]))
    c.exit_bc = int(cfg["exit_bc"])
    _fill_body(c.body, dict(cfg, kind=cfg["body_kind"]))
    parts = cfg.get("parts") or []
    c.nextra = len(parts)
    for e, pd in enumerate(parts):
        _fill_body(c.extra[e], pd)
        c.extra_op[e] = 1 if pd.get("op", "+") == "-" else 0
    for k in ("max_levels", "smooth_iters", "max_vcycles", "fixed_vcycles"):
        setattr(c.mg, k, int(cfg[k]))
    c.mg.tol = float(cfg["tol"])
    c.precision = int(cfg.get("precision", 0))
    if cfg.get("tangent"):                                 # ("nu" | "U" | "R" | "spin" | "amp" | "centre", index)
        name, idx = cfg["tangent"]
        c.tangent_param, c.tangent_index = SEEDS[name], int(idx)
    for k, v in (cfg.get("tune") or {}).items():          # wl_tuning: implementation switches, all zero by default
        if not hasattr(c.tune, k):
            raise KeyError(f"wl_tuning has no field {k}")
        setattr(c.tune, k, int(v))
    return c


def workspace_bytes(cfg: dict) -> int:
    c = make_config(cfg)
    return int(load().wl_workspace_bytes(C.byref(c)))


class WLError(RuntimeError):
    pass


STATIC_MAX_CELLS = 64 * 1024 * 1024       # WL_STATIC_MAX_CELLS of include/wl.h


def energy_static(u, out, dims=None, stream=None):
    """wl_energy_static: (kinetic energy, enstrophy) of a velocity field WITH its ghost layer, written into `out`; allocates
    nothing (the reduction scratch is a static device array of libwl: calls that overlap on the GPU race on it).
    u: torch cuda float32, contiguous, shape (nd, [n2+2,] n1+2, n0+2); out: torch cuda float64 with 2 elements; dims: interior cells
    (n0, n1[, n2]), taken from u.shape when None; stream: a torch stream (None: the current one).  Asynchronous."""
    import torch
    if not (u.is_cuda and u.dtype == torch.float32 and u.is_contiguous()):
        raise TypeError("u must be a contiguous float32 cuda tensor")
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 2):
        raise TypeError("out must be a contiguous float64 cuda tensor with two elements")
    nd = int(u.shape[0])
    if dims is None:
        dims = tuple(int(n) - 2 for n in reversed(u.shape[1:]))
    d = (C.c_int * 3)(*(list(dims) + [1] * (3 - len(dims))))
    st = (stream if stream is not None else torch.cuda.current_stream(u.device)).cuda_stream
    err = C.create_string_buffer(512)
    with torch.cuda.device(u.device):
        rc = load().wl_energy_static(C.c_void_p(u.data_ptr()), nd, d, C.c_void_p(st), C.c_void_p(out.data_ptr()), err, 512)
    if rc != 0:
        raise WLError(f"libwl error {rc}: {err.value.decode()}")
    return out


class Sim:
    """One simulation handle.  Device memory comes from torch; all compute is in libwl."""

    def __init__(self, cfg: dict, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("libwl needs a CUDA device (sm_100a); there is no CPU fallback")
        self._L = load()
        self.cfg = dict(cfg)
        self._c = make_config(cfg)
        self.nd = int(cfg["ndim"])
        self.dims = tuple(int(x) for x in cfg["dims"][: self.nd])
        self.shape = tuple(reversed(self.dims))                 # ([Nz,] Ny, Nx)
        self.ncell = int(np.prod(self.dims))
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        nbytes = int(self._L.wl_workspace_bytes(C.byref(self._c)))
        if nbytes == 0:
            raise WLError("invalid config")
        self.workspace_bytes = nbytes
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self._ws.data_ptr()
        self._base = (base + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self._L.wl_sim_create(C.byref(self._c), C.c_void_p(self._base), C.c_size_t(nbytes),
                                   C.c_void_p(self._stream.cuda_stream), C.byref(h))
        if rc != WL_OK:
            raise WLError(f"wl_sim_create failed: {rc}")
        self._h = h

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            self._L.wl_sim_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, allow=()):
        if rc < 0 and rc not in allow:
            raise WLError(f"libwl error {rc}: {self._L.wl_last_error(self._h).decode()}")
        return rc

    @staticmethod
    def _ptr(a):
        """(pointer, on_device) of a torch tensor or numpy array (fp32, contiguous)."""
        if a is None:
            return None, 0
        if isinstance(a, np.ndarray):
            assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
            return C.c_void_p(a.ctypes.data), 0
        assert a.dtype.is_floating_point and a.element_size() == 4 and a.is_contiguous()
        return C.c_void_p(a.data_ptr()), 1 if a.is_cuda else 0

    # -- the C ABI, same names
    def set_fields(self, u=None, p=None):
        pu, du = self._ptr(u)
        pp, dp = self._ptr(p)
        dev = du if u is not None else dp
        if u is not None and p is not None:
            assert du == dp
        self._chk(self._L.wl_set_fields(self._h, pu, pp, dev))

    def init_tgv(self, sign=1):
        self._chk(self._L.wl_init_tgv(self._h, int(sign)))

    def measure(self, t: float):
        self._chk(self._L.wl_measure(self._h, float(t)))

    def mom_step(self, dt: float):
        self._chk(self._L.wl_mom_step(self._h, float(dt)))

    def step(self, t: float, dt: float, adaptive: bool = False):
        self._chk(self._L.wl_step(self._h, float(t), float(dt), int(adaptive)))

    def cfl(self) -> float:
        out = C.c_float()
        self._chk(self._L.wl_cfl(self._h, C.byref(out)), allow=(WL_ENOCONV,))
        return float(out.value)

    def pressure_force(self, t: float = math.nan) -> np.ndarray:
        F = (C.c_float * 3)()
        self._chk(self._L.wl_pressure_force(self._h, float(t), F))
        return np.array([F[0], F[1], F[2]], dtype=np.float64)

    def energy(self) -> np.ndarray:
        """(kinetic energy, enstrophy) of the current velocity, grid units"""
        out = (C.c_double * 2)()
        self._chk(self._L.wl_energy(self._h, out))
        return np.array([out[0], out[1]])

    # -- fp64 / tangent modes (cfg["precision"] = 1 or cfg["tangent"] = (parameter, index)): the generic engine
    def fields_f64(self, tangent: bool = False):
        """(u, p) as float64 numpy arrays: the values, or (tangent mode) their derivatives d/d(theta)"""
        u = np.empty((self.nd,) + self.shape, dtype=np.float64)
        p = np.empty(self.shape, dtype=np.float64)
        self._chk(self._L.wl_get_fields_f64(self._h, C.c_void_p(u.ctypes.data), C.c_void_p(p.ctypes.data), int(tangent), 0))
        return u, p

    def set_fields_f64(self, u=None, p=None):
        u = None if u is None else np.ascontiguousarray(u, dtype=np.float64)
        p = None if p is None else np.ascontiguousarray(p, dtype=np.float64)
        self._chk(self._L.wl_set_fields_f64(self._h, None if u is None else C.c_void_p(u.ctypes.data),
                                            None if p is None else C.c_void_p(p.ctypes.data), 0))

    def pressure_force_f64(self, t: float = math.nan):
        F, dF = (C.c_double * 3)(), (C.c_double * 3)()
        self._chk(self._L.wl_pressure_force_f64(self._h, float(t), F, dF))
        return np.array(list(F)), np.array(list(dF))

    def energy_f64(self):
        e, de = (C.c_double * 2)(), (C.c_double * 2)()
        self._chk(self._L.wl_energy_f64(self._h, e, de))
        return np.array(list(e)), np.array(list(de))

    def dbg_get_f64(self, name: str, level: int = 0, tangent: bool = False) -> np.ndarray:
        ld = self.level_dims(level if name in ("L", "iD", "x", "r") else 0)
        ncomp = {"u": self.nd, "mu0": self.nd, "L": self.nd, "V": self.nd, "mu1": self.nd * self.nd}.get(name, 1)
        out = np.empty((ncomp,) + tuple(reversed(ld)), dtype=np.float64)
        self._chk(self._L.wl_dbg_get_f64(self._h, name.encode(), int(level), int(tangent), C.c_void_p(out.ctypes.data), C.c_size_t(out.size)))
        return out

    def get_fields(self, u=None, p=None, mu0=None):
        """Copy into the given buffers (torch cuda / torch cpu / numpy); all on the same side."""
        ptrs, devs = [], []
        for a in (u, p, mu0):
            q, d = self._ptr(a)
            ptrs.append(q)
            if a is not None:
                devs.append(d)
        assert len(set(devs)) <= 1
        self._chk(self._L.wl_get_fields(self._h, ptrs[0], ptrs[1], ptrs[2], devs[0] if devs else 0))

    def fields(self):
        """Convenience: (u, p) as float32 numpy arrays, u: (nd, [Nz,] Ny, Nx)."""
        u = np.empty((self.nd,) + self.shape, dtype=np.float32)
        p = np.empty(self.shape, dtype=np.float32)
        self.get_fields(u=u, p=p)
        return u, p

    def stats(self) -> dict:
        st = Stats()
        self._chk(self._L.wl_stats(self._h, C.byref(st)))
        return {"vcycles": [st.vcycles[0], st.vcycles[1]], "res": [st.res[0], st.res[1]],
                "nlevels": st.nlevels, "kernel_launches": st.kernel_launches, "nan_flag": st.nan_flag, "noconv": st.noconv}

    def prof_enable(self, enable: bool = True):
        self._chk(self._L.wl_prof_enable(self._h, int(enable)))

    def prof_read(self) -> dict:
        """{kernel class: (total ms, launches)} since prof_enable; classes never launched are omitted."""
        out = {}
        cls = 0
        while True:
            name = C.create_string_buffer(48)
            ms, n = C.c_double(), C.c_int()
            rc = self._chk(self._L.wl_prof_read(self._h, cls, name, 48, C.byref(ms), C.byref(n)))
            if rc == 1:
                return out
            if n.value:
                out[name.value.decode()] = (ms.value, n.value)
            cls += 1

    def synchronize(self):
        self._stream.synchronize()

    # -- stage hooks (parity tests)
    def level_dims(self, level: int):
        d = (C.c_int * 3)()
        self._chk(self._L.wl_level_dims(self._h, int(level), d))
        return tuple(d[: self.nd])

    def dbg_get(self, name: str, level: int = 0, padded: bool = False) -> np.ndarray:
        ld = self.level_dims(level if name in ("L", "iD", "x", "r", "e", "q") else 0)
        if padded:
            ld = tuple(n + 2 for n in ld)
        ncomp = {"u": self.nd, "u0": self.nd, "mu0": self.nd, "L": self.nd, "V": self.nd, "mu1": self.nd * self.nd}.get(name, 1)
        out = np.empty((ncomp,) + tuple(reversed(ld)), dtype=np.float32)
        fn = self._L.wl_dbg_get_padded if padded else self._L.wl_dbg_get
        self._chk(fn(self._h, name.encode(), int(level), C.c_void_p(out.ctypes.data), C.c_size_t(out.size)))
        return out

    def dbg_set(self, name: str, arr, level: int = 0):
        a = np.ascontiguousarray(arr, dtype=np.float32)
        self._chk(self._L.wl_dbg_set(self._h, name.encode(), int(level), C.c_void_p(a.ctypes.data), C.c_size_t(a.size)))

    def dbg_save_u0(self):
        self._chk(self._L.wl_dbg_save_u0(self._h))

    def dbg_conv_diff_bdim(self, dt, corrector=0):
        self._chk(self._L.wl_dbg_conv_diff_bdim(self._h, float(dt), int(corrector)))

    def dbg_bc(self):
        self._chk(self._L.wl_dbg_bc(self._h))

    def dbg_exit_bc(self, dt):
        self._chk(self._L.wl_dbg_exit_bc(self._h, float(dt)))

    def dbg_project(self, w, dt):
        self._chk(self._L.wl_dbg_project(self._h, float(w), float(dt)), allow=(WL_ENOCONV,))

    def dbg_residual(self):
        self._chk(self._L.wl_dbg_residual(self._h))

    def dbg_apply_gradient(self):
        self._chk(self._L.wl_dbg_apply_gradient(self._h))

    def dbg_restrict(self, level):
        self._chk(self._L.wl_dbg_restrict(self._h, int(level)))

    def dbg_prolong(self, level):
        self._chk(self._L.wl_dbg_prolong(self._h, int(level)))

    def dbg_smooth(self, level, iters):
        self._chk(self._L.wl_dbg_smooth(self._h, int(level), int(iters)))

    def dbg_vcycle(self, level=0):
        self._chk(self._L.wl_dbg_vcycle(self._h, int(level)))

    def dbg_coarse_prog(self, ops):
        """ops: sequence of (kind, level, iters); see wl_dbg_coarse_prog in include/wl.h."""
        n = len(ops)
        A = C.c_int * n
        self._chk(self._L.wl_dbg_coarse_prog(self._h, n, A(*[int(o[0]) for o in ops]), A(*[int(o[1]) for o in ops]),
                                             A(*[int(o[2]) for o in ops])))

    def dbg_pcg_scalars(self, level):
        out = (C.c_double * 8)()
        self._chk(self._L.wl_dbg_pcg_scalars(self._h, int(level), out))
        return dict(zip(("rho", "gamma", "alpha", "beta", "rho0", "rsum", "nlive", "live"), [float(v) for v in out]))
