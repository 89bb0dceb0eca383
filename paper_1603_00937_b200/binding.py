"""Thin Python binding of the C ABI in include/gbe.h (same names, argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs inside libgbe.so.
There is no CPU fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgbe.so")

GBE_MAX_ITERS = 1024
EXPORTS = [
    "gbe_build_graph", "gbe_graph_get_info", "gbe_graph_export", "gbe_density", "gbe_gather", "gbe_sp2",
    "gbe_scatter", "gbe_read_log", "gbe_density_host", "gbe_free_graph", "gbe_strerror", "gbe_last_cuda_error",
    "gbe_version", "gbe_build_graph_host", "gbe_density_timed", "gbe_launch_count", "gbe_density_preset", "gbe_expectation", "gbe_update_graph", "gbe_density_fermi",
    "gbe_graph_set_sp2_path", "gbe_error_norms", "gbe_graph_set_gather_path", "gbe_graph_set_scatter_path", "gbe_set_build_scratch_limit",
    "gbe_set_packed_max_m", "gbe_expectation_static", "gbe_set_dependent_launch",
]


class GbeError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"gbe status {status}: {text}")
        self.status = status


class _CsrView(C.Structure):
    _fields_ = [("n", C.c_int64), ("nnz", C.c_int64), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("val", C.c_void_p)]


class _GraphOpts(C.Structure):
    _fields_ = [("tau", C.c_double), ("power", C.c_int32), ("check_symmetry", C.c_int32)]


class _GraphInfo(C.Structure):
    _fields_ = [("n", C.c_int64), ("nnz_S", C.c_int64), ("n_part", C.c_int64), ("sum_m", C.c_int64),
                ("max_m", C.c_int64), ("nnz_D", C.c_int64), ("dense_elems", C.c_int64), ("n_tiles", C.c_int64),
                ("sp2_flops_per_iter", C.c_double), ("sp2_exec_flops_per_iter", C.c_double),
                ("n_tiles_last", C.c_int64), ("sp2_flops_last_iter", C.c_double),
                ("sp2_exec_flops_last_iter", C.c_double),
                ("eps_min", C.c_double), ("eps_max", C.c_double),
                ("contiguous_cores", C.c_int32), ("tile", C.c_int32), ("workspace_bytes", C.c_size_t),
                ("workspace_bytes_fermi", C.c_size_t), ("resident_sp2", C.c_int32), ("resident_fits", C.c_int32),
                ("resident_cluster", C.c_int32), ("sp2_path_chosen", C.c_int32), ("sp2_sym_flops_per_iter", C.c_double),
                ("n_small", C.c_int64), ("n_bins", C.c_int64), ("workspace_bytes_preset_min", C.c_size_t),
                ("x2_tma", C.c_int32), ("reserved2_", C.c_int32)]


class _Sp2Log(C.Structure):
    _fields_ = [("iters_done", C.c_int32), ("branch", C.c_void_p), ("t1", C.c_void_p), ("t2", C.c_void_p)]


class _PhaseTimes(C.Structure):
    _fields_ = [("bounds_ms", C.c_float), ("bounds_launches", C.c_int32), ("gather_ms", C.c_float),
                ("gather_launches", C.c_int32), ("x2_ms", C.c_float), ("x2_launches", C.c_int32),
                ("trace_ms", C.c_float), ("trace_launches", C.c_int32), ("scatter_ms", C.c_float),
                ("scatter_launches", C.c_int32), ("total_ms", C.c_float), ("x2_last_ms", C.c_float),
                ("x2_last_launches", C.c_int32)]


_lib = None


def lib() -> C.CDLL:
    """Loads libgbe.so (built in-tree by `python -m paper_1603_00937_b200.build`). Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1603_00937_b200.build` "
                              "(there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        for name in ("gbe_strerror", "gbe_last_cuda_error", "gbe_version"):
            getattr(l, name).restype = C.c_char_p
        l.gbe_free_graph.restype = None
        l.gbe_free_graph.argtypes = [C.c_void_p]
        l.gbe_build_graph.argtypes = [C.POINTER(_CsrView), C.POINTER(_GraphOpts), C.c_void_p, C.c_int32, C.c_void_p,
                                      C.POINTER(C.c_void_p)]
        l.gbe_update_graph.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CsrView), C.POINTER(_GraphOpts), C.c_void_p,
                                       C.c_int32, C.c_void_p, C.POINTER(C.c_void_p)]
        l.gbe_graph_get_info.argtypes = [C.c_void_p, C.POINTER(_GraphInfo)]
        l.gbe_graph_export.argtypes = [C.c_void_p] * 9
        l.gbe_density.argtypes = [C.POINTER(_CsrView), C.c_void_p, C.c_double, C.c_int32, C.c_double, C.c_void_p,
                                  C.c_size_t, C.c_void_p, C.c_void_p, C.POINTER(_Sp2Log)]
        l.gbe_density_host.argtypes = l.gbe_density.argtypes
        l.gbe_density_timed.argtypes = l.gbe_density.argtypes + [C.POINTER(_PhaseTimes)]
        l.gbe_build_graph_host.argtypes = l.gbe_build_graph.argtypes
        l.gbe_density_preset.argtypes = [C.POINTER(_CsrView), C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p,
                                         C.c_size_t, C.c_void_p, C.c_void_p, C.POINTER(_Sp2Log)]
        l.gbe_density_fermi.argtypes = [C.POINTER(_CsrView), C.c_void_p, C.c_double, C.c_double, C.c_int32, C.c_void_p,
                                        C.c_size_t, C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]
        l.gbe_expectation.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CsrView), C.c_void_p, C.POINTER(C.c_double)]
        l.gbe_error_norms.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.POINTER(C.c_double)]
        l.gbe_graph_set_sp2_path.argtypes = [C.c_void_p, C.c_int32]
        l.gbe_graph_set_gather_path.argtypes = [C.c_void_p, C.c_int32]
        l.gbe_graph_set_scatter_path.argtypes = [C.c_void_p, C.c_int32]
        l.gbe_set_build_scratch_limit.restype = C.c_size_t
        l.gbe_set_build_scratch_limit.argtypes = [C.c_size_t]
        l.gbe_expectation_static.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_CsrView), C.c_void_p, C.c_void_p]
        l.gbe_set_dependent_launch.restype = C.c_int32
        l.gbe_set_dependent_launch.argtypes = [C.c_int32]
        l.gbe_set_packed_max_m.restype = C.c_int32
        l.gbe_set_packed_max_m.argtypes = [C.c_int32]
        l.gbe_launch_count.restype = C.c_uint64
        l.gbe_launch_count.argtypes = []
        l.gbe_gather.argtypes = [C.POINTER(_CsrView), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        l.gbe_sp2.argtypes = [C.c_void_p, C.c_double, C.c_int32, C.c_double, C.c_void_p, C.c_size_t, C.c_void_p]
        l.gbe_scatter.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p]
        l.gbe_read_log.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(_Sp2Log)]
        _lib = l
    return _lib


def _check(status: int) -> None:
    if status != 0:
        raise GbeError(status, lib().gbe_strerror(status).decode())


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _ptr(t) -> int | None:
    return None if t is None else int(t.data_ptr())


@dataclass
class DeviceCSR:
    """CSR on the device, dtypes of gbe_csr_view."""
    n: int
    row_ptr: torch.Tensor  # int64
    col_idx: torch.Tensor  # int32
    val: torch.Tensor  # float64

    @staticmethod
    def from_host(h, device="cuda") -> "DeviceCSR":
        return DeviceCSR(int(h.n), torch.from_numpy(np.ascontiguousarray(h.row_ptr, dtype=np.int64)).to(device),
                         torch.from_numpy(np.ascontiguousarray(h.col_idx, dtype=np.int32)).to(device),
                         torch.from_numpy(np.ascontiguousarray(h.val, dtype=np.float64)).to(device))

    def view(self) -> _CsrView:
        assert self.row_ptr.dtype == torch.int64 and self.col_idx.dtype == torch.int32 and self.val.dtype == torch.float64
        assert self.row_ptr.is_cuda and self.row_ptr.is_contiguous() and self.col_idx.is_contiguous() and self.val.is_contiguous()
        return _CsrView(self.n, int(self.col_idx.numel()), _ptr(self.row_ptr), _ptr(self.col_idx), _ptr(self.val))


@dataclass
class Sp2Log:
    iters_done: int
    branch: np.ndarray
    t1: np.ndarray
    t2: np.ndarray


class Graph:
    """Owner of an opaque gbe_graph handle."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)
        self._info = None

    @property
    def info(self) -> dict:
        """gbe_graph_info as a dict, read on first use (a build + density loop that never looks at it does not pay for it)."""
        if self._info is None:
            info = _GraphInfo()
            _check(lib().gbe_graph_get_info(self.handle, C.byref(info)))
            self._info = {k: getattr(info, k) for k, _ in _GraphInfo._fields_}
        return self._info

    @property
    def handle(self):
        if not self._h:
            raise ValueError("graph already freed")
        return self._h

    def free(self):
        if self._h:
            lib().gbe_free_graph(self._h)
            self._h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def new_workspace(self, device="cuda") -> torch.Tensor:
        return torch.empty(self.info["workspace_bytes"], dtype=torch.uint8, device=device)

    def export(self, stream=None) -> dict:
        return gbe_graph_export(self, stream)


def gbe_build_graph(H: DeviceCSR, tau: float, part: torch.Tensor | None, n_part: int, power: int = 2,
                    check_symmetry: bool = False, stream=None) -> Graph:
    opts = _GraphOpts(float(tau), int(power), int(bool(check_symmetry)))
    if part is not None:
        assert part.dtype == torch.int32 and part.is_cuda and part.is_contiguous() and part.numel() == H.n
    out = C.c_void_p()
    v = H.view()
    _check(lib().gbe_build_graph(C.byref(v), C.byref(opts), _ptr(part), int(n_part), _stream(stream), C.byref(out)))
    return Graph(out.value)


def gbe_build_graph_host(H_host, tau: float, part_host: np.ndarray | None, n_part: int, power: int = 2,
                         check_symmetry: bool = False, stream=None) -> Graph:
    """H_host: numpy fields n, row_ptr (int64), col_idx (int32), val (float64); part_host: int32[n] or None. HOST memory."""
    opts = _GraphOpts(float(tau), int(power), int(bool(check_symmetry)))
    rp = np.ascontiguousarray(H_host.row_ptr, dtype=np.int64)
    ci = np.ascontiguousarray(H_host.col_idx, dtype=np.int32)
    va = np.ascontiguousarray(H_host.val, dtype=np.float64)
    pt = None if part_host is None else np.ascontiguousarray(part_host, dtype=np.int32)
    v = _CsrView(int(H_host.n), int(ci.size), rp.ctypes.data, ci.ctypes.data, va.ctypes.data)
    out = C.c_void_p()
    _check(lib().gbe_build_graph_host(C.byref(v), C.byref(opts), None if pt is None else pt.ctypes.data, int(n_part),
                                      _stream(stream), C.byref(out)))
    return Graph(out.value)


def gbe_update_graph(prev: Graph, D_prev: torch.Tensor, H: DeviceCSR, tau: float, part: torch.Tensor | None, n_part: int,
                     stream=None) -> Graph:
    """Eq.(8): the graph of the next MD step from D(t - dt) (on prev's pattern) and H(t), symbolic square."""
    assert D_prev.dtype == torch.float64 and D_prev.is_cuda and D_prev.numel() == prev.info["nnz_D"]
    opts = _GraphOpts(float(tau), 0, 0)
    if part is not None:
        assert part.dtype == torch.int32 and part.is_cuda and part.is_contiguous() and part.numel() == H.n
    out = C.c_void_p()
    v = H.view()
    _check(lib().gbe_update_graph(prev.handle, _ptr(D_prev), C.byref(v), C.byref(opts), _ptr(part), int(n_part),
                                  _stream(stream), C.byref(out)))
    return Graph(out.value)


def gbe_graph_set_sp2_path(g: "Graph", path: int) -> None:
    """0 auto, 1 tiled kernels, 2 shared-memory-resident kernel, 3 packed kernel for the small communities (include/gbe.h)."""
    _check(lib().gbe_graph_set_sp2_path(g._h, int(path)))
    g._info = None  # sp2_path_chosen / resident_sp2 change: read again on next use


def gbe_graph_set_scatter_path(g: "Graph", path: int) -> None:
    """0 auto (bulk copies where the graph allows them), 1 the register variant (include/gbe.h)."""
    _check(lib().gbe_graph_set_scatter_path(g._h, int(path)))


def gbe_graph_set_gather_path(g: "Graph", path: int) -> None:
    """0 auto, 1 staged through a shared-memory row buffer, 2 direct to global memory (include/gbe.h)."""
    _check(lib().gbe_graph_set_gather_path(g._h, int(path)))


def gbe_set_build_scratch_limit(nbytes: int) -> int:
    """Scratch limit of the graph builds for the candidate bitmaps (include/gbe.h); returns the previous limit."""
    return int(lib().gbe_set_build_scratch_limit(int(nbytes)))


def gbe_set_dependent_launch(on: bool) -> bool:
    """Programmatic dependent launch of the SP2 kernels on / off (process-wide); returns the previous setting."""
    return bool(lib().gbe_set_dependent_launch(1 if on else 0))


def gbe_set_packed_max_m(m: int) -> int:
    """Largest community the packed SP2 kernel takes in graphs built from now on (include/gbe.h); returns the previous value."""
    old = int(lib().gbe_set_packed_max_m(int(m)))
    if old < 0:
        raise GbeError(-1, "gbe_set_packed_max_m: out of range")
    return old


def gbe_launch_count() -> int:
    return int(lib().gbe_launch_count())


def gbe_graph_export(g: Graph, stream=None) -> dict:
    i = g.info
    dev = "cuda"
    out = dict(
        S_row_ptr=torch.empty(i["n"] + 1, dtype=torch.int64, device=dev),
        S_col=torch.empty(i["nnz_S"], dtype=torch.int32, device=dev),
        sub_ptr=torch.empty(i["n_part"] + 1, dtype=torch.int64, device=dev),
        sub_idx=torch.empty(i["sum_m"], dtype=torch.int32, device=dev),
        ncore=torch.empty(i["n_part"], dtype=torch.int32, device=dev),
        D_row_ptr=torch.empty(i["n"] + 1, dtype=torch.int64, device=dev),
        D_col=torch.empty(i["nnz_D"], dtype=torch.int32, device=dev),
    )
    _check(lib().gbe_graph_export(g.handle, _stream(stream), *[_ptr(out[k]) for k in
                                  ("S_row_ptr", "S_col", "sub_ptr", "sub_idx", "ncore", "D_row_ptr", "D_col")]))
    return out


def _new_log(iters: int):
    br = np.zeros(max(iters, 1), dtype=np.uint8)
    t1 = np.zeros(iters + 1, dtype=np.float64)
    t2 = np.zeros(iters + 1, dtype=np.float64)
    return _Sp2Log(0, br.ctypes.data, t1.ctypes.data, t2.ctypes.data), (br, t1, t2)


def _finish_log(clog, arrs) -> Sp2Log:
    k = int(clog.iters_done)
    br, t1, t2 = arrs
    return Sp2Log(k, br[:k].copy(), t1[:k + 1].copy(), t2[:k + 1].copy())


def gbe_density(H: DeviceCSR, g: Graph, n_occ: float, iters: int, idem_tol: float = -1.0,
                workspace: torch.Tensor | None = None, D_val: torch.Tensor | None = None, want_log: bool = True,
                stream=None):
    """Returns (D_val, Sp2Log | None).  With want_log the call synchronises the stream to read the log."""
    if workspace is None:
        workspace = g.new_workspace()
    if D_val is None:
        D_val = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
    v = H.view()
    clog, arrs = _new_log(iters) if want_log else (None, None)
    _check(lib().gbe_density(C.byref(v), g.handle, float(n_occ), int(iters), float(idem_tol), _ptr(workspace),
                             workspace.numel(), _stream(stream), _ptr(D_val), C.byref(clog) if want_log else None))
    return D_val, (_finish_log(clog, arrs) if want_log else None)


def gbe_density_timed(H: DeviceCSR, g: Graph, n_occ: float, iters: int, idem_tol: float = -1.0,
                      workspace: torch.Tensor | None = None, D_val: torch.Tensor | None = None, stream=None):
    """gbe_density with one CUDA-event pair per launch; synchronises.  Returns (D_val, dict of gbe_phase_times)."""
    if workspace is None:
        workspace = g.new_workspace()
    if D_val is None:
        D_val = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
    v = H.view()
    pt = _PhaseTimes()
    _check(lib().gbe_density_timed(C.byref(v), g.handle, float(n_occ), int(iters), float(idem_tol), _ptr(workspace),
                                   workspace.numel(), _stream(stream), _ptr(D_val), None, C.byref(pt)))
    return D_val, {k: getattr(pt, k) for k, _ in _PhaseTimes._fields_}


def gbe_density_preset(H: DeviceCSR, g: Graph, branch, trace_every_iteration: bool = True,
                       workspace: torch.Tensor | None = None, D_val: torch.Tensor | None = None, want_log: bool = True,
                       stream=None):
    """gbe_density with a pre-determined SP2 sequence: branch[k] in {0, 1}, host array.  Returns (D_val, log)."""
    if workspace is None:
        workspace = g.new_workspace()
    if D_val is None:
        D_val = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
    br = np.ascontiguousarray(branch, dtype=np.uint8)
    iters = int(br.size)
    v = H.view()
    clog, arrs = _new_log(iters) if want_log else (None, None)
    _check(lib().gbe_density_preset(C.byref(v), g.handle, br.ctypes.data if iters else None, iters,
                                    int(bool(trace_every_iteration)), _ptr(workspace), workspace.numel(), _stream(stream),
                                    _ptr(D_val), C.byref(clog) if want_log else None))
    return D_val, (_finish_log(clog, arrs) if want_log else None)


def gbe_density_fermi(H: DeviceCSR, g: Graph, mu: float, beta: float, order: int, workspace: torch.Tensor | None = None,
                      D_val: torch.Tensor | None = None, want_n_elec: bool = True, stream=None):
    """Finite-temperature D by the Chebyshev Fermi-operator expansion (Eq.(7)).  Returns (D_val, n_elec | None)."""
    if workspace is None:
        workspace = torch.empty(g.info["workspace_bytes_fermi"], dtype=torch.uint8, device="cuda")
    if D_val is None:
        D_val = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
    v = H.view()
    ne = C.c_double(0.0)
    _check(lib().gbe_density_fermi(C.byref(v), g.handle, float(mu), float(beta), int(order), _ptr(workspace),
                                   workspace.numel(), _stream(stream), _ptr(D_val), C.byref(ne) if want_n_elec else None))
    return D_val, (float(ne.value) if want_n_elec else None)


def gbe_expectation(g: Graph, D_val: torch.Tensor, A: DeviceCSR, stream=None) -> float:
    """<A> = Tr[D A]; A = H gives the band energy.  Synchronises."""
    assert D_val.dtype == torch.float64 and D_val.is_cuda and D_val.numel() == g.info["nnz_D"]
    v = A.view()
    out = C.c_double(0.0)
    _check(lib().gbe_expectation(g.handle, _ptr(D_val), C.byref(v), _stream(stream), C.byref(out)))
    return float(out.value)


GBE_STATIC_MAX_N = 131072  # gbe.h


def gbe_expectation_static(g: Graph, D_val: torch.Tensor, A: DeviceCSR, out: torch.Tensor, stream=None) -> torch.Tensor:
    """<A> = Tr[D A] into the caller's DEVICE double `out` without any allocation or synchronisation (scratch: a static
    1 MiB device array inside the library, n <= GBE_STATIC_MAX_N; calls that overlap on the GPU race on it)."""
    assert D_val.dtype == torch.float64 and D_val.is_cuda and D_val.numel() == g.info["nnz_D"]
    assert out.dtype == torch.float64 and out.is_cuda and out.numel() >= 1 and out.is_contiguous()
    v = A.view()
    _check(lib().gbe_expectation_static(g.handle, _ptr(D_val), C.byref(v), _stream(stream), _ptr(out)))
    return out


def gbe_error_norms(g: Graph, D_val: torch.Tensor, D_ref: torch.Tensor, stream=None) -> tuple[float, float, float]:
    """(max error over the stored entries, sum of squared errors over them, ||D - D_ref||_F^2 over the full matrix)
    against a dense n x n reference on the device (Fig.2).  Synchronises."""
    n = g.info["n"]
    assert D_val.dtype == torch.float64 and D_val.is_cuda and D_val.numel() == g.info["nnz_D"]
    assert D_ref.dtype == torch.float64 and D_ref.is_cuda and D_ref.dim() == 2 and D_ref.shape[0] == n
    assert D_ref.stride(1) == 1 and D_ref.stride(0) >= n and D_ref.shape[1] == n
    out = (C.c_double * 3)()
    _check(lib().gbe_error_norms(g.handle, _ptr(D_val), _ptr(D_ref), int(D_ref.stride(0)), _stream(stream), out))
    return float(out[0]), float(out[1]), float(out[2])


def gbe_gather(H: DeviceCSR, g: Graph, workspace: torch.Tensor, stream=None) -> None:
    v = H.view()
    _check(lib().gbe_gather(C.byref(v), g.handle, _ptr(workspace), workspace.numel(), _stream(stream)))


def gbe_sp2(g: Graph, n_occ: float, iters: int, idem_tol: float, workspace: torch.Tensor, stream=None) -> None:
    _check(lib().gbe_sp2(g.handle, float(n_occ), int(iters), float(idem_tol), _ptr(workspace), workspace.numel(),
                         _stream(stream)))


def gbe_scatter(g: Graph, workspace: torch.Tensor, D_val: torch.Tensor, stream=None) -> None:
    _check(lib().gbe_scatter(g.handle, _ptr(workspace), workspace.numel(), _stream(stream), _ptr(D_val)))


def gbe_read_log(g: Graph, workspace: torch.Tensor, iters: int = GBE_MAX_ITERS, stream=None) -> Sp2Log:
    clog, arrs = _new_log(iters)
    _check(lib().gbe_read_log(g.handle, _ptr(workspace), workspace.numel(), _stream(stream), C.byref(clog)))
    return _finish_log(clog, arrs)


def gbe_density_host(H_host, g: Graph, n_occ: float, iters: int, idem_tol: float = -1.0,
                     workspace: torch.Tensor | None = None, D_val_host: np.ndarray | None = None,
                     want_log: bool = False, stream=None):
    """H_host: object with numpy fields n, row_ptr (int64), col_idx (int32), val (float64) - HOST memory
    (pinned or pageable).  Copies in, runs, copies D back, synchronises.  H_host=None reuses the device copy of H that
    gbe_build_graph_host left with the graph."""
    if workspace is None:
        workspace = g.new_workspace()
    if D_val_host is None:
        D_val_host = np.empty(g.info["nnz_D"], dtype=np.float64)
    if H_host is not None:
        rp = np.ascontiguousarray(H_host.row_ptr, dtype=np.int64)
        ci = np.ascontiguousarray(H_host.col_idx, dtype=np.int32)
        va = np.ascontiguousarray(H_host.val, dtype=np.float64)
        v = _CsrView(int(H_host.n), int(ci.size), rp.ctypes.data, ci.ctypes.data, va.ctypes.data)
    clog, arrs = _new_log(iters) if want_log else (None, None)
    _check(lib().gbe_density_host(C.byref(v) if H_host is not None else None, g.handle, float(n_occ), int(iters), float(idem_tol), _ptr(workspace),
                                  workspace.numel(), _stream(stream), D_val_host.ctypes.data,
                                  C.byref(clog) if want_log else None))
    return D_val_host, (_finish_log(clog, arrs) if want_log else None)
