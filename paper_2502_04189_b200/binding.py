"""Thin ctypes binding of libfizzy.so (include/fizzy.h): same entry-point names, argument
marshalling only.  PyTorch is used for device memory (the workspace tensor) and the stream.

Importing this module loads the CUDA library and raises if it is missing: there is no CPU
fallback and nothing here imports the oracle."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfizzy.so")

FIZZY_OK, FIZZY_EINVAL, FIZZY_ENOMEM, FIZZY_ECUDA, FIZZY_ESTATE, FIZZY_ENOCONV = range(6)
_STATUS = {0: "FIZZY_OK", 1: "FIZZY_EINVAL", 2: "FIZZY_ENOMEM", 3: "FIZZY_ECUDA", 4: "FIZZY_ESTATE", 5: "FIZZY_ENOCONV"}

EXPORTS = ["fizzy_workspace_bytes", "fizzy_create", "fizzy_destroy", "fizzy_set_fields",
           "fizzy_rk3_substep", "fizzy_poisson_solve", "fizzy_get_fields", "fizzy_gamma", "fizzy_diagnostics",
           "fizzy_launch_count", "fizzy_last_error", "fizzy_timing_enable", "fizzy_timing_get",
           "fizzy_rk3_step", "fizzy_graph_enable", "fizzy_stable_dt", "fizzy_check_finite",
           "fizzy_varcoef_workspace_bytes", "fizzy_poisson_solve_varcoef", "fizzy_set_pressure_solver",
           "fizzy_count_nonfinite_static", "fizzy_abi_version"]


class FizzyGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
                ("zf", C.POINTER(C.c_double))]


class FizzyBC(C.Structure):
    _fields_ = [("z_wall", C.c_int), ("t_wall", C.c_double * 2)]


class FizzyProps(C.Structure):
    _fields_ = [("rho", C.c_double * 2), ("mu", C.c_double * 2), ("kth", C.c_double * 2),
                ("cp", C.c_double * 2), ("sigma", C.c_double), ("eps", C.c_double),
                ("delta", C.c_double), ("gamma_rel", C.c_double), ("gamma_abs", C.c_double),
                ("g", C.c_double * 3), ("rho_ref", C.c_double), ("beta", C.c_double),
                ("t_ref", C.c_double), ("force", C.c_double * 3), ("lin_forcing", C.c_double),
                ("heat", C.c_int)]


class FizzyError(RuntimeError):
    def __init__(self, status, text=""):
        super().__init__("%s%s" % (_STATUS.get(status, status), (": " + text) if text else ""))
        self.status = status


def load_library(path: str = LIB_PATH) -> C.CDLL:
    if not os.path.exists(path):
        raise ImportError("libfizzy.so is missing at %s: run `python -m paper_2502_04189_b200.build` "
                          "(there is no CPU fallback)" % path)
    lib = C.CDLL(path)
    vp, dp = C.c_void_p, C.c_void_p  # field pointers are passed as raw addresses (host or device)
    lib.fizzy_workspace_bytes.restype = C.c_size_t
    lib.fizzy_workspace_bytes.argtypes = [C.POINTER(FizzyGrid), C.POINTER(FizzyBC), C.POINTER(FizzyProps)]
    lib.fizzy_create.restype = C.c_int
    lib.fizzy_create.argtypes = [C.POINTER(FizzyGrid), C.POINTER(FizzyBC), C.POINTER(FizzyProps),
                                 vp, C.c_size_t, vp, C.POINTER(vp)]
    lib.fizzy_destroy.restype = C.c_int
    lib.fizzy_destroy.argtypes = [vp]
    lib.fizzy_set_fields.restype = C.c_int
    lib.fizzy_set_fields.argtypes = [vp] + [dp] * 7
    lib.fizzy_get_fields.restype = C.c_int
    lib.fizzy_get_fields.argtypes = [vp] + [dp] * 7
    lib.fizzy_rk3_substep.restype = C.c_int
    lib.fizzy_rk3_substep.argtypes = [vp, C.c_int, C.c_double]
    lib.fizzy_poisson_solve.restype = C.c_int
    lib.fizzy_poisson_solve.argtypes = [vp, dp, dp]
    lib.fizzy_varcoef_workspace_bytes.restype = C.c_size_t
    lib.fizzy_varcoef_workspace_bytes.argtypes = [vp]
    lib.fizzy_poisson_solve_varcoef.restype = C.c_int
    lib.fizzy_poisson_solve_varcoef.argtypes = [vp, dp, dp, dp, vp, C.c_size_t, C.c_double, C.c_int,
                                                C.POINTER(C.c_int), C.POINTER(C.c_double)]
    lib.fizzy_set_pressure_solver.restype = C.c_int
    lib.fizzy_set_pressure_solver.argtypes = [vp, C.c_int, vp, C.c_size_t, C.c_double, C.c_int]
    lib.fizzy_diagnostics.restype = C.c_int
    lib.fizzy_diagnostics.argtypes = [vp, C.POINTER(C.c_double)]
    lib.fizzy_rk3_step.restype = C.c_int
    lib.fizzy_rk3_step.argtypes = [vp, C.c_double]
    lib.fizzy_graph_enable.restype = C.c_int
    lib.fizzy_graph_enable.argtypes = [vp, C.c_int]
    lib.fizzy_stable_dt.restype = C.c_int
    lib.fizzy_stable_dt.argtypes = [vp, C.c_double, C.POINTER(C.c_double)]
    lib.fizzy_check_finite.restype = C.c_int
    lib.fizzy_check_finite.argtypes = [vp, C.POINTER(C.c_longlong)]
    lib.fizzy_count_nonfinite_static.restype = C.c_int
    lib.fizzy_count_nonfinite_static.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_longlong, vp, C.POINTER(C.c_longlong),
                                                 C.c_char_p, C.c_size_t]
    lib.fizzy_abi_version.restype = C.c_int
    lib.fizzy_abi_version.argtypes = []
    lib.fizzy_gamma.restype = C.c_double
    lib.fizzy_gamma.argtypes = [vp]
    lib.fizzy_launch_count.restype = C.c_longlong
    lib.fizzy_launch_count.argtypes = [vp]
    lib.fizzy_timing_enable.restype = C.c_int
    lib.fizzy_timing_enable.argtypes = [vp, C.c_int]
    lib.fizzy_timing_get.restype = C.c_int
    lib.fizzy_timing_get.argtypes = [vp, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_double),
                                     C.POINTER(C.c_longlong), C.c_int]
    lib.fizzy_last_error.restype = C.c_char_p
    lib.fizzy_last_error.argtypes = [vp]
    return lib


_lib = load_library()
FIZZY_ABI_VERSION = 3   # the version this binding was written against (include/fizzy.h)
if _lib.fizzy_abi_version() != FIZZY_ABI_VERSION:
    raise ImportError("libfizzy.so has interface version %d, this binding expects %d: rebuild with "
                      "`python -m paper_2502_04189_b200.build`" % (_lib.fizzy_abi_version(), FIZZY_ABI_VERSION))


def structs_from_cfg(cfg: dict):
    """cfg: the plain dict of paper_2502_04189_b200.workloads (keys nx..t_top, optional zf)."""
    g = FizzyGrid(cfg["nx"], cfg["ny"], cfg["nz"], cfg["lx"], cfg["ly"], cfg["lz"], None)
    keep = None
    if cfg.get("zf") is not None:
        keep = np.ascontiguousarray(cfg["zf"], dtype=np.float64)
        g.zf = keep.ctypes.data_as(C.POINTER(C.c_double))
    bc = FizzyBC(int(cfg.get("z_wall", 0)), (C.c_double * 2)(cfg.get("t_bot", 0.0), cfg.get("t_top", 0.0)))
    pr = FizzyProps()
    pr.rho[:] = [cfg["rho1"], cfg["rho2"]]
    pr.mu[:] = [cfg["mu1"], cfg["mu2"]]
    pr.kth[:] = [cfg.get("k1", 1.0), cfg.get("k2", 1.0)]
    pr.cp[:] = [cfg.get("cp1", 1.0), cfg.get("cp2", 1.0)]
    pr.sigma, pr.eps, pr.delta = cfg.get("sigma", 0.0), cfg["eps"], cfg.get("delta", 1e-100)
    pr.gamma_rel, pr.gamma_abs = cfg.get("gamma_rel", 0.0), cfg.get("gamma_abs", 0.0)
    pr.g[:] = [cfg.get("gx", 0.0), cfg.get("gy", 0.0), cfg.get("gz", 0.0)]
    pr.rho_ref, pr.beta, pr.t_ref = cfg.get("rho_ref", 0.0), cfg.get("beta", 0.0), cfg.get("t_ref", 0.0)
    pr.force[:] = [cfg.get("fx", 0.0), cfg.get("fy", 0.0), cfg.get("fz", 0.0)]
    pr.lin_forcing = cfg.get("a_lin", 0.0)
    pr.heat = int(cfg.get("heat", 0))
    return g, bc, pr, keep


def _addr(a):
    """Raw address of a torch tensor (host or device), a numpy array, an int, or None."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.dtype.is_floating_point and a.element_size() == 8 and a.is_contiguous()
    return a.data_ptr()


def fizzy_workspace_bytes(cfg: dict) -> int:
    g, bc, pr, _keep = structs_from_cfg(cfg)
    return int(_lib.fizzy_workspace_bytes(C.byref(g), C.byref(bc), C.byref(pr)))


FIZZY_STATIC_MAX_VALUES = 1 << 27
FIZZY_STATIC_MAX_FIELDS = 8


def fizzy_count_nonfinite_static(fields, n=None, stream=None) -> int:
    """Number of Inf / NaN values in up to 8 device fields, with no context and no allocation on the library's side
    (the scratch is an array built into libfizzy.so; see include/fizzy.h for who needs that and for the size limit).
    `fields`: CUDA tensors of float64 (or raw device addresses, then `n` = values per field is required).  Marshalling
    only: the addresses go into a ctypes array, the library does the rest.  Run with the fields' device current."""
    ptrs = [_addr(a) for a in fields]
    if n is None:
        n = fields[0].numel() if fields else 0
        assert all(a.numel() == n for a in fields), "fields of different sizes: pass n"
    arr = (C.c_void_p * max(len(ptrs), 1))(*ptrs)
    cnt, err = C.c_longlong(-1), C.create_string_buffer(512)
    st = _lib.fizzy_count_nonfinite_static(arr, len(ptrs), int(n), stream.cuda_stream if stream is not None else None,
                                           C.byref(cnt), err, len(err))
    if st != FIZZY_OK:
        raise FizzyError(st, err.value.decode())
    return cnt.value


class Fizzy:
    """One solver context on the current CUDA device.  Field arguments are torch tensors
    (cuda or cpu/pinned) or numpy arrays of shape (nz, ny, nx), float64, contiguous."""

    def __init__(self, cfg: dict, stream=None, device="cuda:0"):
        import torch  # device memory + stream only
        if not torch.cuda.is_available():
            raise FizzyError(FIZZY_ECUDA, "no CUDA device: libfizzy has no CPU fallback")
        self._torch = torch
        self.cfg = dict(cfg)
        self.shape = (cfg["nz"], cfg["ny"], cfg["nx"])
        self.heat = bool(cfg.get("heat", 0))
        self.device = torch.device(device)
        g, bc, pr, keep = structs_from_cfg(cfg)
        nbytes = int(_lib.fizzy_workspace_bytes(C.byref(g), C.byref(bc), C.byref(pr)))
        if nbytes == 0:
            raise FizzyError(FIZZY_EINVAL, "invalid grid / bc / props")
        self.workspace_bytes = nbytes
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) & ~255
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            st = _lib.fizzy_create(C.byref(g), C.byref(bc), C.byref(pr), aligned, nbytes,
                                   self.stream.cuda_stream, C.byref(h))
        self._h = h if h.value else None
        self._check(st)

    def _on_device(self):
        """The library launches on the CURRENT device: make the context's device current around every call."""
        return self._torch.cuda.device(self.device)

    def _check(self, st):
        if st != FIZZY_OK:
            text = _lib.fizzy_last_error(self._h).decode() if self._h else ""
            raise FizzyError(st, text)

    def close(self):
        h = getattr(self, "_h", None)
        if h:
            self._h = None
            try:
                with self._on_device():
                    _lib.fizzy_destroy(h)
            except Exception:   # called from __del__ at interpreter shutdown with torch already torn down: the process is ending
                pass

    __del__ = close

    # ---- the C-ABI calls, same names ----
    def fizzy_set_fields(self, u=None, v=None, w=None, p=None, phi=None, T=None, p_prev=None):
        with self._on_device():
            self._check(_lib.fizzy_set_fields(self._h, *[_addr(a) for a in (u, v, w, p, phi, T, p_prev)]))

    def fizzy_get_fields(self, u=None, v=None, w=None, p=None, phi=None, T=None, p_prev=None):
        with self._on_device():
            self._check(_lib.fizzy_get_fields(self._h, *[_addr(a) for a in (u, v, w, p, phi, T, p_prev)]))

    def fizzy_rk3_substep(self, stage: int, dt: float):
        with self._on_device():
            self._check(_lib.fizzy_rk3_substep(self._h, int(stage), float(dt)))

    def fizzy_poisson_solve(self, rhs, p):
        with self._on_device():
            self._check(_lib.fizzy_poisson_solve(self._h, _addr(rhs), _addr(p)))

    def fizzy_poisson_solve_varcoef(self, rhs, p, phi=None, rtol=1e-10, max_iter=100):
        """Returns (iterations, relative residual).  The scratch tensor is torch-owned and kept for later calls."""
        with self._on_device():
            nbytes = _lib.fizzy_varcoef_workspace_bytes(self._h)
            if getattr(self, "_vc_work", None) is None or self._vc_work.numel() < nbytes:
                self._vc_work = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
            it, rr = C.c_int(), C.c_double()
            self._check(_lib.fizzy_poisson_solve_varcoef(self._h, _addr(rhs), _addr(phi), _addr(p),
                                                         self._vc_work.data_ptr(), nbytes, float(rtol), int(max_iter),
                                                         C.byref(it), C.byref(rr)))
        return it.value, rr.value

    def fizzy_set_pressure_solver(self, solver: int, rtol=1e-12, max_iter=200):
        """solver 1 = the variable-coefficient multigrid path; the scratch tensor is torch-owned and kept alive here."""
        with self._on_device():
            ptr, nbytes = None, 0
            if solver == 1:
                nbytes = _lib.fizzy_varcoef_workspace_bytes(self._h)
                if getattr(self, "_ps_work", None) is None or self._ps_work.numel() < nbytes:
                    self._ps_work = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
                ptr = self._ps_work.data_ptr()
            self._check(_lib.fizzy_set_pressure_solver(self._h, int(solver), ptr, nbytes, float(rtol), int(max_iter)))

    def fizzy_diagnostics(self) -> np.ndarray:
        out = (C.c_double * 8)()
        with self._on_device():
            self._check(_lib.fizzy_diagnostics(self._h, out))
        return np.array(out[:])

    def fizzy_rk3_step(self, dt: float):
        with self._on_device():
            self._check(_lib.fizzy_rk3_step(self._h, float(dt)))

    def fizzy_graph_enable(self, on: bool):
        self._check(_lib.fizzy_graph_enable(self._h, int(bool(on))))

    def fizzy_stable_dt(self, cfl: float = 0.5) -> float:
        dt = C.c_double()
        with self._on_device():
            self._check(_lib.fizzy_stable_dt(self._h, float(cfl), C.byref(dt)))
        return dt.value

    def fizzy_check_finite(self) -> int:
        n = C.c_longlong()
        with self._on_device():
            self._check(_lib.fizzy_check_finite(self._h, C.byref(n)))
        return n.value

    def fizzy_gamma(self) -> float:
        with self._on_device():
            return float(_lib.fizzy_gamma(self._h))

    def fizzy_launch_count(self) -> int:
        return int(_lib.fizzy_launch_count(self._h))

    def fizzy_timing_enable(self, on: bool):
        self._check(_lib.fizzy_timing_enable(self._h, int(bool(on))))

    def fizzy_timing_get(self, reset: bool = False) -> dict:
        """{kernel name: (total ms, launches)} for every kernel slot with at least one launch."""
        out, i = {}, 0
        while True:
            name, ms, n = C.c_char_p(), C.c_double(), C.c_longlong()
            if _lib.fizzy_timing_get(self._h, i, C.byref(name), C.byref(ms), C.byref(n), int(reset)) != FIZZY_OK:
                break
            if n.value:
                out[name.value.decode()] = (ms.value, n.value)
            i += 1
        return out

    # ---- conveniences (marshalling only) ----
    def step(self, dt: float):
        self.fizzy_rk3_step(dt)

    def set_fields_numpy(self, **f):
        self.fizzy_set_fields(**{k: np.ascontiguousarray(a, dtype=np.float64) for k, a in f.items()})
        self.stream.synchronize()

    def get_fields_numpy(self) -> dict:
        names = ["u", "v", "w", "p", "phi", "p_prev"] + (["T"] if self.heat else [])
        out = {n: np.empty(self.shape) for n in names}
        self.fizzy_get_fields(**out)
        self.stream.synchronize()
        return out
