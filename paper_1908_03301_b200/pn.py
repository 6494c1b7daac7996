"""Thin Python binding of the C-ABI library `libpn.so` (include/pn.h) -- argument marshalling only.

Every step of the path runs inside the library's CUDA kernels.  PyTorch is used for exactly three
things: allocating device memory (the workspace, inputs, outputs), naming the CUDA stream, and
moving numpy inputs to the device.  There is no CPU fallback: if `libpn.so` is missing or no CUDA
device is present, creating a `Network` raises.

    net = Network(nx, ny, nz)              # pn_create (workspace = a torch uint8 tensor)
    net.set_conductances(gx, gy, gz)       # pn_set_conductances (numpy / torch CPU / torch CUDA)
    info = net.solve(direction=0, tol=1e-10)   # pn_solve
    P = net.pressures()                    # pn_get_pressures -> torch.float64 CUDA tensor (nz, ny, nx)
    q_in, q_out, g_eff, k_eff = net.flux() # pn_flux
    net.close()                            # pn_destroy
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpn.so")

PN_OK, PN_NO_SPANNING_CLUSTER, PN_MAX_ITERS = 0, 1, 2
PN_ERR_ARG, PN_ERR_STATE, PN_ERR_VALUE, PN_ERR_WORKSPACE, PN_ERR_CUDA, PN_ERR_BREAKDOWN = -1, -2, -3, -4, -5, -6
PN_ERR_TOO_LARGE = -7
PN_NOALLOC_MAX_NODES = 1 << 28
(PN_OPT_MAX_ITERS, PN_OPT_DELTA, PN_OPT_X0, PN_OPT_CHUNK, PN_OPT_SKIP_LABEL, PN_OPT_KERNEL, PN_OPT_PROFILE,
 PN_OPT_PEEL, PN_OPT_LATERAL, PN_OPT_GRAPH, PN_OPT_XDEFER, PN_OPT_REUSE_LABELS, PN_OPT_COMPACT, PN_OPT_CONTRACT,
 PN_OPT_TILE) = range(15)
CLASS_INLET, CLASS_OUTLET, CLASS_SOLVED, CLASS_INLET_ONLY, CLASS_OUTLET_ONLY, CLASS_FLOATING = range(6)

# every symbol include/pn.h declares (tests check that the library exports each of them)
SYMBOLS = ("pn_workspace_bytes", "pn_create", "pn_set_conductances", "pn_solve", "pn_get_pressures",
           "pn_get_classes", "pn_flux", "pn_set_option", "pn_launch_count", "pn_destroy", "pn_strerror",
           "pn_last_error", "pn_residual_history", "pn_dissipation", "pn_update_conductances",
           "pn_replace_conductances", "pn_dissipation_noalloc")


class PnInfo(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int), ("outer_cycles", ctypes.c_int), ("inner_iters", ctypes.c_int),
                ("kernel_scheme", ctypes.c_int), ("rel_residual", ctypes.c_double), ("b_norm", ctypes.c_double),
                ("n_solved", ctypes.c_longlong), ("n_inlet_only", ctypes.c_longlong),
                ("n_outlet_only", ctypes.c_longlong), ("n_floating", ctypes.c_longlong),
                ("t_label_ms", ctypes.c_double), ("t_solve_ms", ctypes.c_double),
                ("t_stencil_ms", ctypes.c_double), ("t_update_ms", ctypes.c_double),
                ("n_timed_iters", ctypes.c_int), ("n_xskip", ctypes.c_int),
                ("n_peeled", ctypes.c_longlong), ("n_unknowns", ctypes.c_longlong),
                ("n_chain", ctypes.c_longlong), ("n_long_rows", ctypes.c_longlong), ("labels_reused", ctypes.c_int),
                ("residual_recovered", ctypes.c_int)]


@dataclass
class SolveInfo:
    status: int
    outer_cycles: int
    inner_iters: int
    rel_residual: float
    b_norm: float
    n_solved: int
    n_inlet_only: int
    n_outlet_only: int
    n_floating: int
    t_label_ms: float
    t_solve_ms: float
    t_stencil_ms: float = 0.0
    t_update_ms: float = 0.0
    n_timed_iters: int = 0
    kernel_scheme: int = 0
    n_peeled: int = 0
    n_xskip: int = 0
    labels_reused: int = 0
    n_unknowns: int = 0
    n_chain: int = 0
    n_long_rows: int = 0
    residual_recovered: int = 0


class PnError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libpn error {code}: {text}")
        self.code = code


_lib = None


def load_library(path: str = LIB_PATH) -> ctypes.CDLL:
    """dlopen libpn.so and declare the prototypes of include/pn.h.  Raises if it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not built: run `python -m paper_1908_03301_b200.build` "
                                "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, cp = ctypes.c_void_p, ctypes.c_char_p
    dp = ctypes.POINTER(ctypes.c_double)
    lib.pn_workspace_bytes.argtypes = [ctypes.c_int] * 3
    lib.pn_workspace_bytes.restype = ctypes.c_size_t
    lib.pn_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp,
                              ctypes.c_size_t]
    lib.pn_create.restype = ctypes.c_int
    lib.pn_set_conductances.argtypes = [vp, vp, vp, vp, ctypes.c_int]
    lib.pn_set_conductances.restype = ctypes.c_int
    lib.pn_update_conductances.argtypes = [vp, ctypes.c_longlong, vp, vp, vp, ctypes.c_int]
    lib.pn_update_conductances.restype = ctypes.c_int
    lib.pn_replace_conductances.argtypes = [vp, vp, vp, vp, ctypes.c_int]
    lib.pn_replace_conductances.restype = ctypes.c_int
    lib.pn_solve.argtypes = [vp, ctypes.c_int, ctypes.c_double, ctypes.POINTER(PnInfo)]
    lib.pn_solve.restype = ctypes.c_int
    lib.pn_get_pressures.argtypes = [vp, vp, ctypes.c_int]
    lib.pn_get_pressures.restype = ctypes.c_int
    lib.pn_get_classes.argtypes = [vp, vp, ctypes.c_int]
    lib.pn_get_classes.restype = ctypes.c_int
    lib.pn_flux.argtypes = [vp, dp, dp, dp, dp]
    lib.pn_flux.restype = ctypes.c_int
    lib.pn_set_option.argtypes = [vp, ctypes.c_int, ctypes.c_double]
    lib.pn_set_option.restype = ctypes.c_int
    lib.pn_launch_count.argtypes = [vp]
    lib.pn_launch_count.restype = ctypes.c_longlong
    lib.pn_dissipation.argtypes = [vp, dp]
    lib.pn_dissipation.restype = ctypes.c_int
    lib.pn_dissipation_noalloc.argtypes = [ctypes.c_int] * 3 + [vp, vp, vp, vp, ctypes.c_int, vp, ctypes.c_int, vp]
    lib.pn_dissipation_noalloc.restype = ctypes.c_int
    lib.pn_residual_history.argtypes = [vp, dp, ctypes.c_int]
    lib.pn_residual_history.restype = ctypes.c_int
    lib.pn_destroy.argtypes = [vp]
    lib.pn_destroy.restype = ctypes.c_int
    lib.pn_strerror.argtypes = [ctypes.c_int]
    lib.pn_strerror.restype = cp
    lib.pn_last_error.argtypes = [vp]
    lib.pn_last_error.restype = cp
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load_library().pn_strerror(code).decode()


class Network:
    """One bond network on one CUDA device (wraps a `pn_ctx*`)."""

    def __init__(self, nx: int, ny: int, nz: int = 1, device: int = 0, stream=None):
        import torch
        self._torch = torch
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        if not torch.cuda.is_available():
            raise RuntimeError("libpn needs a CUDA device (no CPU fallback)")
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.device = torch.device("cuda", device)
        nbytes = self._lib.pn_workspace_bytes(self.nx, self.ny, self.nz)
        if nbytes == 0:
            raise PnError(PN_ERR_ARG, "bad lattice shape")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self._lib.pn_create(ctypes.byref(self._h), self.nx, self.ny, self.nz, device,
                                 ctypes.c_void_p(self.stream.cuda_stream), ctypes.c_void_p(self.workspace.data_ptr()),
                                 nbytes)
        if rc != PN_OK:
            self._h = ctypes.c_void_p()
            raise PnError(rc, strerror(rc))

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, rc: int, ok=(PN_OK,)):
        if rc not in ok:
            extra = self._lib.pn_last_error(self._h).decode() if self._h else ""
            raise PnError(rc, strerror(rc) + (f" [{extra}]" if extra else ""))
        return rc

    @property
    def n_nodes(self) -> int:
        return self.nx * self.ny * self.nz

    def set_option(self, key: int, value: float):
        self._check(self._lib.pn_set_option(self._h, key, float(value)))

    # -- S0 --------------------------------------------------------------------------------------
    def set_conductances(self, gx, gy, gz=None, _entry="pn_set_conductances"):
        """gx, gy, gz: numpy float32 arrays / torch tensors of nx*ny*nz entries (shape (nz, ny, nx))."""
        torch = self._torch
        import numpy as np
        keep = []
        ptrs = []
        on_device = None
        for g in (gx, gy, gz):
            if g is None:
                ptrs.append(None)
                continue
            if isinstance(g, torch.Tensor):
                t = g.detach()
                if t.dtype != torch.float32 or not t.is_contiguous():
                    t = t.to(torch.float32).contiguous()
                dev = t.is_cuda
                ptr = t.data_ptr()
            else:
                t = np.ascontiguousarray(g, dtype=np.float32)
                dev = False
                ptr = t.ctypes.data
            n = t.numel() if isinstance(t, torch.Tensor) else t.size
            if n != self.n_nodes:
                raise PnError(PN_ERR_ARG, "conductance array has the wrong number of entries")
            if on_device is None:
                on_device = dev
            elif on_device != dev:
                raise PnError(PN_ERR_ARG, "mix of host and device conductance arrays")
            keep.append(t)
            ptrs.append(ctypes.c_void_p(ptr))
        rc = getattr(self._lib, _entry)(self._h, ptrs[0], ptrs[1], ptrs[2], 1 if on_device else 0)
        del keep
        self._check(rc)

    def replace_conductances(self, gx, gy, gz=None):
        """pn_replace_conductances: new values for all bonds of the network the handle holds (labels and warm start kept
        when no bond crosses zero).  Arguments as set_conductances."""
        self.set_conductances(gx, gy, gz, _entry="pn_replace_conductances")

    def update_conductances(self, axis, node, value):
        """pn_update_conductances: sparse update.  axis (int32), node (int64), value (float32): numpy arrays or torch
        tensors of equal length, all on the host or all on the device."""
        torch = self._torch
        import numpy as np
        want = (("int32", torch.int32), ("int64", torch.int64), ("float32", torch.float32))
        keep, ptrs, dev = [], [], None
        for a, (npd, td) in zip((axis, node, value), want):
            if isinstance(a, torch.Tensor):
                t = a.detach().to(td).contiguous()
                d, ptr, n = t.is_cuda, t.data_ptr(), t.numel()
            else:
                t = np.ascontiguousarray(a, dtype=npd)
                d, ptr, n = False, t.ctypes.data, t.size
            if dev is None:
                dev, count = d, n
            elif dev != d or n != count:
                raise PnError(PN_ERR_ARG, "update lists differ in length or in where they live")
            keep.append(t)
            ptrs.append(ctypes.c_void_p(ptr))
        rc = self._lib.pn_update_conductances(self._h, count, ptrs[0], ptrs[1], ptrs[2], 1 if dev else 0)
        del keep
        self._check(rc)

    # -- S1..S7 ----------------------------------------------------------------------------------
    def solve(self, direction: int = 0, tol: float = 1e-10, accept=(PN_OK, PN_NO_SPANNING_CLUSTER)) -> SolveInfo:
        info = PnInfo()
        rc = self._lib.pn_solve(self._h, int(direction), float(tol), ctypes.byref(info))
        self._check(rc, ok=tuple(accept))
        return SolveInfo(rc, info.outer_cycles, info.inner_iters, info.rel_residual, info.b_norm, info.n_solved,
                         info.n_inlet_only, info.n_outlet_only, info.n_floating, info.t_label_ms, info.t_solve_ms,
                         info.t_stencil_ms, info.t_update_ms, info.n_timed_iters, info.kernel_scheme, info.n_peeled, info.n_xskip,
                         info.labels_reused, info.n_unknowns, info.n_chain, info.n_long_rows, info.residual_recovered)

    def pressures(self, out=None):
        """fp64 pressures on all nodes as a CUDA tensor of shape (nz, ny, nx)."""
        torch = self._torch
        if out is None:
            out = torch.empty((self.nz, self.ny, self.nx), dtype=torch.float64, device=self.device)
        self._check(self._lib.pn_get_pressures(self._h, ctypes.c_void_p(out.data_ptr()), 1 if out.is_cuda else 0))
        return out

    def pressures_host(self, out=None):
        """fp64 pressures copied straight into a host numpy array (device->host inside the C call)."""
        import numpy as np
        if out is None:
            out = np.empty((self.nz, self.ny, self.nx), dtype=np.float64)
        self._check(self._lib.pn_get_pressures(self._h, ctypes.c_void_p(out.ctypes.data), 0))
        return out

    def classes(self):
        torch = self._torch
        out = torch.empty((self.nz, self.ny, self.nx), dtype=torch.int8, device=self.device)
        self._check(self._lib.pn_get_classes(self._h, ctypes.c_void_p(out.data_ptr()), 1))
        return out

    # -- S8 --------------------------------------------------------------------------------------
    def flux(self):
        v = [ctypes.c_double() for _ in range(4)]
        self._check(self._lib.pn_flux(self._h, *[ctypes.byref(x) for x in v]))
        return tuple(x.value for x in v)

    def residual_history(self):
        """True fp64 relative residuals of the last solve, one per residual evaluation (first = initial guess)."""
        n = self._lib.pn_residual_history(self._h, None, 0)
        if n < 0:
            self._check(n)
        buf = (ctypes.c_double * max(n, 1))()
        self._lib.pn_residual_history(self._h, buf, n)
        return [buf[i] for i in range(n)]

    def dissipation(self) -> float:
        """G_E = sum over all bonds g (dP_bond)^2: the effective conductance with an error quadratic in that of P."""
        v = ctypes.c_double()
        self._check(self._lib.pn_dissipation(self._h, ctypes.byref(v)))
        return v.value

    def launch_count(self) -> int:
        return int(self._lib.pn_launch_count(self._h))

    def close(self):
        if self._h:
            self._lib.pn_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def dissipation_noalloc(gx, gy, gz, pressures, out, periodic_mask: int = 0, stream=None) -> None:
    """pn_dissipation_noalloc: G_E of the network the CALLER holds, written to `out[0]` on the stream; allocates nothing.

    gx, gy, gz (None for 2D): float32 CUDA tensors of shape (nz, ny, nx) as given to `Network.set_conductances`;
    `pressures`: float64 CUDA tensor of that shape (`Network.pressures()`); `out`: float64 CUDA tensor with >= 1 element,
    allocated by the caller.  Only enqueues: read `out` after synchronising the stream.  At most PN_NOALLOC_MAX_NODES
    nodes (PnError with PN_ERR_TOO_LARGE beyond); overlapping calls on one GPU share one scratch array and race."""
    import torch
    lib = load_library()
    for name, t, dt in (("gx", gx, torch.float32), ("gy", gy, torch.float32), ("gz", gz, torch.float32),
                        ("pressures", pressures, torch.float64), ("out", out, torch.float64)):
        if t is None and name == "gz":
            continue
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dt and t.is_contiguous()):
            raise TypeError(f"{name}: contiguous CUDA tensor of {dt} expected")
    if pressures.dim() != 3 or out.numel() < 1:
        raise ValueError("pressures: shape (nz, ny, nx); out: at least one element")
    nz, ny, nx = pressures.shape
    for name, t in (("gx", gx), ("gy", gy), ("gz", gz)):
        if t is not None and t.numel() != pressures.numel():
            raise ValueError(f"{name}: {pressures.numel()} elements expected")
    if stream is None:
        stream = torch.cuda.current_stream(pressures.device)
    rc = lib.pn_dissipation_noalloc(nx, ny, nz, gx.data_ptr(), gy.data_ptr(), gz.data_ptr() if gz is not None else None,
                                    pressures.data_ptr(), int(periodic_mask), out.data_ptr(), pressures.device.index,
                                    ctypes.c_void_p(stream.cuda_stream))
    if rc != PN_OK:
        raise PnError(rc, strerror(rc))
