"""ctypes binding of the fp64 CPU oracle (oracle/wl_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA
package (paper_2407_16032_b200) and shares no code with it.

The shared library is compiled on first use for the CPU it runs on (-march=native), into
oracle/_build/, keyed by a hash of the source and of the host's CPU flags, so a library
built on one machine is never executed on another.
"""
from __future__ import annotations

import ctypes as C
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "wl_oracle.c"

BODY_NONE, BODY_SPHERE, BODY_TORUS, BODY_CYLINDER, BODY_PLANE = 0, 1, 2, 3, 4
MOTION_STATIC, MOTION_SIN = 0, 1


class Part(C.Structure):
    _fields_ = [
        ("kind", C.c_int), ("centre", C.c_double * 3), ("R", C.c_double), ("r", C.c_double), ("axis", C.c_int),
        ("motion", C.c_int), ("amp", C.c_double * 3), ("freq", C.c_double * 3), ("phase", C.c_double * 3),
        ("shell", C.c_double), ("scale_amp", C.c_double * 3), ("scale_freq", C.c_double), ("scale_phase", C.c_double),
        ("spin", C.c_double), ("op", C.c_int),
    ]


class Config(C.Structure):
    _fields_ = [
        ("ndim", C.c_int), ("dims", C.c_int * 3),
        ("L", C.c_double), ("U", C.c_double * 3), ("nu", C.c_double),
        ("periodic", C.c_int * 3), ("exit_bc", C.c_int),
        ("eps", C.c_double),
        ("dt0", C.c_double), ("dt_max", C.c_double), ("cfl_c", C.c_double), ("cfl_cnu", C.c_double),
        ("body_kind", C.c_int), ("centre", C.c_double * 3), ("R", C.c_double), ("r", C.c_double),
        ("axis", C.c_int), ("motion", C.c_int),
        ("amp", C.c_double * 3), ("freq", C.c_double * 3), ("phase", C.c_double * 3),
        ("max_levels", C.c_int), ("smooth_iters", C.c_int), ("max_vcycles", C.c_int),
        ("fixed_vcycles", C.c_int), ("tol", C.c_double),
        ("shell", C.c_double), ("scale_amp", C.c_double * 3), ("scale_freq", C.c_double), ("scale_phase", C.c_double),
        ("spin", C.c_double), ("nextra", C.c_int), ("extra", Part * 3),
    ]


def _cpu_key() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha1((flags + _SRC.read_text()).encode()).hexdigest()[:12]


def build(verbose: bool = False) -> Path:
    """Compile oracle/wl_oracle.c for this host; returns the .so path."""
    out_dir = _HERE / "_build"
    out_dir.mkdir(exist_ok=True)
    so = out_dir / f"libwl_oracle_{_cpu_key()}.so"
    if not so.exists():
        tmp = so.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=gnu11",
               "-o", str(tmp), str(_SRC), "-lm"]
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return so


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        L.wlo_create.restype = C.c_void_p
        L.wlo_create.argtypes = [C.POINTER(Config)]
        L.wlo_destroy.argtypes = [C.c_void_p]
        L.wlo_array.restype = C.POINTER(C.c_double)
        L.wlo_array.argtypes = [C.c_void_p, C.c_char_p, C.c_int, C.POINTER(C.c_int)]
        for name in ("wlo_kernel_K", "wlo_kernel_mu0", "wlo_kernel_mu1"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double, C.c_double]
        L.wlo_quick.restype = C.c_double
        L.wlo_quick.argtypes = [C.c_double] * 3
        L.wlo_body_eval.restype = C.c_double
        L.wlo_body_eval.argtypes = [C.POINTER(Config), C.POINTER(C.c_double), C.c_double,
                                    C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.wlo_measure.argtypes = [C.c_void_p, C.c_double]
        L.wlo_bc.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.wlo_exit_bc.argtypes = [C.c_void_p, C.c_double]
        L.wlo_conv_diff.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.wlo_bdim.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.wlo_smooth.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.wlo_restrict.argtypes = [C.c_void_p, C.c_int]
        L.wlo_prolong_increment.argtypes = [C.c_void_p, C.c_int]
        L.wlo_vcycle.argtypes = [C.c_void_p, C.c_int]
        L.wlo_residual.argtypes = [C.c_void_p]
        L.wlo_solve.restype = C.c_int
        L.wlo_solve.argtypes = [C.c_void_p]
        L.wlo_divergence.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.wlo_project.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.wlo_mom_step.argtypes = [C.c_void_p, C.c_double]
        L.wlo_cfl.restype = C.c_double
        L.wlo_cfl.argtypes = [C.c_void_p]
        L.wlo_pressure_force.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.wlo_init_tgv.argtypes = [C.c_void_p, C.c_int]
        L.wlo_energy.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.wlo_nlevels.restype = C.c_int
        L.wlo_nlevels.argtypes = [C.c_void_p]
        L.wlo_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.wlo_matvec.restype = C.c_double
        L.wlo_matvec.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.wlo_poisson_update.argtypes = [C.c_void_p]
        L.wlo_num_threads.restype = C.c_int
        _lib = L
    return _lib


def wi_motion(cfg: dict):
    """(amp[3], freq[3], phase[3]) of the sinusoidal translation from the plain dict: either three-vectors under
    amp3 / freq3 / phase3, or the scalars amp / freq / phase acting along heave_dir (wl_inputs.CONFIG_DEFAULTS)."""
    if cfg.get("amp3") is not None:
        return ([float(v) for v in cfg["amp3"]], [float(v) for v in cfg["freq3"]], [float(v) for v in cfg["phase3"]])
    a, f, p = [0.0] * 3, [0.0] * 3, [0.0] * 3
    d = int(cfg["heave_dir"])
    a[d], f[d], p[d] = float(cfg["amp"]), float(cfg["freq"]), float(cfg["phase"])
    return a, f, p


def make_config(cfg: dict) -> Config:
    """Build the oracle's POD config from a plain dict (see wl_inputs.CONFIG_DEFAULTS)."""
    c = Config()
    nd = int(cfg["ndim"])
    c.ndim = nd
    for d in range(3):
        c.dims[d] = int(cfg["dims"][d]) if d < nd else 1
        c.U[d] = float(cfg["U"][d]) if d < len(cfg["U"]) else 0.0
        c.periodic[d] = int(cfg["periodic"][d]) if d < nd else 0
        c.centre[d] = float(cfg["centre"][d]) if d < len(cfg["centre"]) else 0.0
    for k in ("L", "nu", "eps", "dt0", "dt_max", "cfl_c", "cfl_cnu", "R", "r", "tol"):
        setattr(c, k, float(cfg[k]))
    amp, freq, phase = wi_motion(cfg)
    for d in range(3):
        c.amp[d], c.freq[d], c.phase[d] = amp[d], freq[d], phase[d]
    for k in ("exit_bc", "body_kind", "axis", "motion", "max_levels", "smooth_iters",
              "max_vcycles", "fixed_vcycles"):
        setattr(c, k, int(cfg[k]))
    # general bodies: shell, diagonal scaling map, spin, further primitives (all optional in the dict)
    c.shell, c.scale_freq, c.scale_phase = float(cfg.get("shell", 0.0)), float(cfg.get("scale_freq", 0.0)), float(cfg.get("scale_phase", 0.0))
    c.spin = float(cfg.get("spin", 0.0))
    for d in range(3):
        c.scale_amp[d] = float((cfg.get("scale_amp") or (0.0, 0.0, 0.0))[d])
    parts = cfg.get("parts") or []
    c.nextra = len(parts)
    for e, pd in enumerate(parts):
        q = c.extra[e]
        full = dict(centre=(0.0, 0.0, 0.0), R=0.0, r=0.0, axis=0, motion=MOTION_STATIC, heave_dir=1, amp=0.0, freq=0.0, phase=0.0,
                    amp3=None, freq3=None, phase3=None, shell=0.0, scale_amp=(0.0, 0.0, 0.0), scale_freq=0.0, scale_phase=0.0,
                    spin=0.0, op="+")
        full.update(pd)
        q.kind, q.R, q.r, q.axis, q.motion = int(full["kind"]), float(full["R"]), float(full["r"]), int(full["axis"]), int(full["motion"])
        amp, freq, phase = wi_motion(full)
        for d in range(3):
            q.centre[d] = float(full["centre"][d]) if d < len(full["centre"]) else 0.0
            q.amp[d], q.freq[d], q.phase[d] = amp[d], freq[d], phase[d]
            q.scale_amp[d] = float(full["scale_amp"][d])
        q.shell, q.scale_freq, q.scale_phase, q.spin = float(full["shell"]), float(full["scale_freq"]), float(full["scale_phase"]), float(full["spin"])
        q.op = 1 if full["op"] == "-" else 0
    return c


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class OracleSim:
    """One oracle simulation.  Arrays are exposed as numpy *views* of the C storage with
    shape (ncomp, S2, S1, S0) (paper-padded: one ghost per side; 2-D has S2 == 1)."""

    def __init__(self, cfg: dict):
        self.cfg = dict(cfg)
        self._c = make_config(cfg)
        self._h = lib().wlo_create(C.byref(self._c))
        if not self._h:
            raise ValueError("oracle: invalid config")
        self.nd = int(cfg["ndim"])
        self.dims = tuple(int(x) for x in cfg["dims"][: self.nd])

    def close(self):
        if self._h:
            lib().wlo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def nlevels(self) -> int:
        return lib().wlo_nlevels(self._h)

    def arr(self, name: str, level: int = 0) -> np.ndarray:
        shape = (C.c_int * 4)()
        p = lib().wlo_array(self._h, name.encode(), level, shape)
        if not p:
            raise KeyError(name)
        shp = tuple(int(x) for x in shape)
        return np.ctypeslib.as_array(p, shape=shp)

    def interior(self, name: str, level: int = 0) -> np.ndarray:
        a = self.arr(name, level)
        if self.nd == 3:
            return a[:, 1:-1, 1:-1, 1:-1]
        return a[:, :, 1:-1, 1:-1]

    # --- state I/O on interior-sized arrays (ncomp, [Nz,] Ny, Nx) -------------------
    def set_fields(self, u=None, p=None):
        if u is not None:
            self.interior("u")[...] = np.asarray(u, dtype=np.float64).reshape(self.interior("u").shape)
            self.bc()
        if p is not None:
            self.interior("p")[...] = np.asarray(p, dtype=np.float64).reshape(self.interior("p").shape)

    # --- stages -----------------------------------------------------------------------
    def measure(self, t: float):
        lib().wlo_measure(self._h, float(t))

    def bc(self):
        lib().wlo_bc(self._h, _dp(self.arr("u")))

    def exit_bc(self, dt):
        lib().wlo_exit_bc(self._h, float(dt))

    def conv_diff(self, w: str = "u"):
        """r = conv_diff(w) stored in the 'f' array."""
        lib().wlo_conv_diff(self._h, _dp(self.arr(w)), _dp(self.arr("f")))

    def bdim(self, dt, corr=0):
        lib().wlo_bdim(self._h, float(dt), int(corr))

    def smooth(self, level, its):
        lib().wlo_smooth(self._h, int(level), int(its))

    def restrict(self, level):
        lib().wlo_restrict(self._h, int(level))

    def prolong_increment(self, level):
        lib().wlo_prolong_increment(self._h, int(level))

    def vcycle(self, level=0):
        lib().wlo_vcycle(self._h, int(level))

    def residual(self):
        lib().wlo_residual(self._h)

    def solve(self) -> int:
        return lib().wlo_solve(self._h)

    def divergence(self) -> np.ndarray:
        out = np.zeros_like(self.arr("p"))
        lib().wlo_divergence(self._h, _dp(out))
        return out

    def project(self, w, dt):
        lib().wlo_project(self._h, float(w), float(dt))

    def mom_step(self, dt):
        lib().wlo_mom_step(self._h, float(dt))

    def cfl(self) -> float:
        return lib().wlo_cfl(self._h)

    def pressure_force(self, t) -> np.ndarray:
        F = np.zeros(3)
        lib().wlo_pressure_force(self._h, float(t), _dp(F))
        return F

    def init_tgv(self, sign=1):
        lib().wlo_init_tgv(self._h, int(sign))

    def energy(self) -> np.ndarray:
        """(kinetic energy, enstrophy): the staggered-grid sums of reading R-E2"""
        out = np.zeros(2)
        lib().wlo_energy(self._h, _dp(out))
        return out

    def matvec(self, level, x: np.ndarray):
        """q = A_level x on padded arrays (ghosts of x are wrapped in place); returns (q, q.x)."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        q = np.zeros_like(x)
        d = lib().wlo_matvec(self._h, int(level), _dp(x), _dp(q))
        return q, d

    def poisson_update(self):
        lib().wlo_poisson_update(self._h)

    def stats(self):
        v = (C.c_int * 2)()
        r = (C.c_double * 2)()
        lib().wlo_stats(self._h, v, r)
        return {"vcycles": [v[0], v[1]], "res": [r[0], r[1]]}


def kernel_K(s, eps):
    return lib().wlo_kernel_K(float(s), float(eps))


def kernel_mu0(d, eps):
    return lib().wlo_kernel_mu0(float(d), float(eps))


def kernel_mu1(d, eps):
    return lib().wlo_kernel_mu1(float(d), float(eps))


def quick(U, Cc, D):
    return lib().wlo_quick(float(U), float(Cc), float(D))


def body_eval(cfg: dict, x, t):
    c = make_config(cfg)
    xp = (C.c_double * 3)(*[float(v) for v in list(x) + [0.0] * (3 - len(x))])
    n = (C.c_double * 3)()
    v = (C.c_double * 3)()
    d = lib().wlo_body_eval(C.byref(c), xp, float(t), n, v)
    return d, np.array(list(n)), np.array(list(v))


def num_threads() -> int:
    return lib().wlo_num_threads()
