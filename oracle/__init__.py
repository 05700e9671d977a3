"""CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT) -- ctypes loader for fizzy_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It shares no code with paper_2502_04189_b200 and never imports it.

`Oracle(cfg)` takes the plain configuration dict produced by the workload generators
(keys listed in `PARAM_KEYS`) and exposes the steps of the RK3 substep of PAPER.md:32-36 as
restated in DESIGN.md; see fizzy_oracle.h for the passages each routine follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fizzy_oracle.c")
_HDR = os.path.join(_HERE, "fizzy_oracle.h")
_LIB = os.path.join(_HERE, "liborc.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP on the outer loops). Returns the .so path."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True, text=True)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
        ("z_wall", C.c_int), ("has_zf", C.c_int),
        ("rho1", C.c_double), ("rho2", C.c_double), ("mu1", C.c_double), ("mu2", C.c_double),
        ("k1", C.c_double), ("k2", C.c_double), ("cp1", C.c_double), ("cp2", C.c_double),
        ("sigma", C.c_double), ("eps", C.c_double), ("delta", C.c_double),
        ("gamma_rel", C.c_double), ("gamma_abs", C.c_double),
        ("gx", C.c_double), ("gy", C.c_double), ("gz", C.c_double),
        ("rho_ref", C.c_double), ("beta", C.c_double), ("t_ref", C.c_double),
        ("fx", C.c_double), ("fy", C.c_double), ("fz", C.c_double),
        ("a_lin", C.c_double), ("heat", C.c_int), ("t_bot", C.c_double), ("t_top", C.c_double),
    ]


PARAM_KEYS = [f[0] for f in _Params._fields_ if f[0] != "has_zf"]

_DEFAULTS = dict(z_wall=0, k1=1.0, k2=1.0, cp1=1.0, cp2=1.0, sigma=0.0, delta=1e-100,
                 gamma_rel=0.0, gamma_abs=0.0, gx=0.0, gy=0.0, gz=0.0, rho_ref=0.0, beta=0.0,
                 t_ref=0.0, fx=0.0, fy=0.0, fz=0.0, a_lin=0.0, heat=0, t_bot=0.0, t_top=0.0)

_lib = None
_dp = C.POINTER(C.c_double)


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.POINTER(_Params), _dp]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_set_fields.argtypes = [C.c_void_p] + [_dp] * 7
        lib.orc_get_fields.argtypes = [C.c_void_p] + [_dp] * 7
        lib.orc_substep.argtypes = [C.c_void_p, C.c_int, C.c_double]
        lib.orc_substep.restype = C.c_int
        lib.orc_poisson_solve.argtypes = [C.c_void_p, _dp, _dp]
        lib.orc_set_solver.argtypes = [C.c_void_p, C.c_int]
        lib.orc_varcoef_solve.argtypes = [C.c_void_p, _dp, _dp]
        lib.orc_varcoef_solve.restype = C.c_int
        lib.orc_diagnostics.argtypes = [C.c_void_p, _dp]
        lib.orc_stable_dt.argtypes = [C.c_void_p, C.c_double]
        lib.orc_stable_dt.restype = C.c_double
        lib.orc_gamma.argtypes = [C.c_void_p]
        lib.orc_gamma.restype = C.c_double
        lib.orc_get_intermediate.argtypes = [C.c_void_p, C.c_char_p, _dp]
        lib.orc_get_intermediate.restype = C.c_int
        lib.orc_momentum_rhs.argtypes = [C.c_void_p, _dp, _dp, _dp]
        lib.orc_phi_rhs.argtypes = [C.c_void_p, C.c_double, _dp]
        lib.orc_temperature_rhs.argtypes = [C.c_void_p, _dp]
        lib.orc_fft.argtypes = [C.c_int, _dp, _dp, C.c_int]
        lib.orc_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_load().orc_num_threads())


def fft(x: np.ndarray, sign: int = -1) -> np.ndarray:
    """The oracle's own radix-2 FFT of a complex vector (power-of-two length)."""
    re = np.ascontiguousarray(np.real(x), dtype=np.float64).copy()
    im = np.ascontiguousarray(np.imag(x), dtype=np.float64).copy()
    _load().orc_fft(len(re), _ptr(re), _ptr(im), sign)
    return re + 1j * im


class Oracle:
    """One solver state.  Arrays are numpy float64 of shape (nz, ny, nx) (x fastest)."""

    def __init__(self, cfg: dict):
        lib = _load()
        self.cfg = dict(_DEFAULTS)
        self.cfg.update({k: v for k, v in cfg.items() if k in PARAM_KEYS or k == "zf"})
        prm = _Params()
        for k in PARAM_KEYS:
            setattr(prm, k, self.cfg[k])
        zf = self.cfg.get("zf")
        self._zf = _c(zf)
        prm.has_zf = 0 if zf is None else 1
        self.shape = (prm.nz, prm.ny, prm.nx)
        self.heat = bool(prm.heat)
        self._h = lib.orc_create(C.byref(prm), _ptr(self._zf))
        if not self._h:
            raise MemoryError("orc_create failed")

    def close(self):
        if getattr(self, "_h", None):
            _load().orc_destroy(self._h)
            self._h = None

    __del__ = close

    def set_fields(self, u, v, w, p, phi, T=None, p_prev=None):
        arrs = [_c(a) for a in (u, v, w, p, phi, T, p_prev)]
        for a in arrs:
            assert a is None or a.shape == self.shape, (a.shape, self.shape)
        _load().orc_set_fields(self._h, *[_ptr(a) for a in arrs])

    def get_fields(self) -> dict:
        names = ["u", "v", "w", "p", "phi", "T", "p_prev"]
        out = {n: np.empty(self.shape) for n in names if n != "T" or self.heat}
        _load().orc_get_fields(self._h, *[_ptr(out.get(n)) for n in names])
        return out

    def substep(self, stage: int, dt: float):
        rc = _load().orc_substep(self._h, int(stage), float(dt))
        if rc != 0:
            raise ValueError("orc_substep: bad arguments or fields not set")

    def step(self, dt: float):
        for s in range(3):
            self.substep(s, dt)

    def poisson_solve(self, rhs) -> np.ndarray:
        rhs = _c(rhs)
        out = np.empty(self.shape)
        _load().orc_poisson_solve(self._h, _ptr(rhs), _ptr(out))
        return out

    def set_solver(self, solver: int):
        """0: the constant-coefficient splitting; 1: the variable-coefficient problem."""
        _load().orc_set_solver(self._h, int(solver))

    def varcoef_solve(self, rhs) -> np.ndarray:
        rhs = _c(rhs)
        out = np.empty(self.shape)
        self.varcoef_iterations = _load().orc_varcoef_solve(self._h, _ptr(rhs), _ptr(out))
        return out

    def diagnostics(self) -> np.ndarray:
        """[volume of fluid 1, kinetic energy, max|u|, max|D(u)|, interfacial area, mean T, Nu bottom, Nu top]"""
        out = np.zeros(8)
        _load().orc_diagnostics(self._h, out.ctypes.data_as(_dp))
        return out

    def stable_dt(self, cfl: float = 0.5) -> float:
        """N16: cfl * min(advective, viscous, capillary, ACDI, thermal limit) of the current fields."""
        return float(_load().orc_stable_dt(self._h, float(cfl)))

    def gamma(self) -> float:
        return float(_load().orc_gamma(self._h))

    def intermediate(self, name: str) -> np.ndarray:
        out = np.empty(self.shape)
        if _load().orc_get_intermediate(self._h, name.encode(), _ptr(out)) != 0:
            raise KeyError(name)
        return out

    def momentum_rhs(self):
        r = [np.empty(self.shape) for _ in range(3)]
        _load().orc_momentum_rhs(self._h, *[_ptr(a) for a in r])
        return r

    def temperature_rhs(self) -> np.ndarray:
        out = np.empty(self.shape)
        _load().orc_temperature_rhs(self._h, _ptr(out))
        return out

    def phi_rhs(self, gamma: float) -> np.ndarray:
        out = np.empty(self.shape)
        _load().orc_phi_rhs(self._h, float(gamma), _ptr(out))
        return out
