"""ctypes binding of include/pnn.h.  Argument marshalling only: every step of the path runs inside libpnn.so.

Pointers: DEVICE arguments are passed as integers (`tensor.data_ptr()`); HOST arguments as C-contiguous
numpy arrays.  `PaiNN` is a small convenience holder (model + workspace) used by the tests and bench.py; it
only allocates output tensors with torch and forwards pointers.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

__all__ = [
    "PNN_OK", "PNN_BF16", "PNN_FP32", "PNN_FP64", "PNN_ENERGY", "PNN_FORCES", "PnnError", "pnn_config", "lib",
    "lib_path", "pnn_status_string", "pnn_last_cuda_error", "pnn_weights_count", "pnn_model_create",
    "pnn_model_destroy", "pnn_branch_mlp_create", "pnn_branch_mlp_destroy", "pnn_branch_weights",
    "pnn_workspace_create", "pnn_workspace_destroy", "pnn_workspace_bytes", "pnn_workspace_edge_tape_bytes",
    "PNN_WS_FORCES", "PNN_WS_NO_EDGE_TAPE", "pnn_build_graph",
    "pnn_graph_view", "pnn_graph_copy", "pnn_build_graph_static", "PNN_STATIC_MAX_ATOMS", "PNN_STATIC_MAX_STRUCTS",
    "PNN_STATIC_MAX_EDGES", "PNN_STATIC_SCRATCH_BYTES", "PNN_STATIC_EDGE_OVERFLOW", "PNN_IMAGES_MINIMUM", "PNN_IMAGES_ALL",
    "pnn_eval", "pnn_eval_replay", "pnn_set_globals", "pnn_eval_blended", "pnn_eval_host", "pnn_stream_create", "pnn_stream_destroy", "pnn_stream_submit", "pnn_stream_wait",
    "pnn_stream_drain", "pnn_stream_launch_count", "pnn_stream_bytes", "pnn_check_async_errors", "pnn_measure_alu_peak", "pnn_measure_l2_peak", "pnn_launch_count", "pnn_profile_enable",
    "pnn_profile_read", "pnn_gemm_bf16",
    "PaiNN", "PRECISIONS",
]

PNN_OK = 0
PNN_BF16, PNN_FP32, PNN_FP64 = 0, 1, 2
PNN_ENERGY, PNN_FORCES = 1, 2
PNN_STATIC_MAX_ATOMS, PNN_STATIC_MAX_STRUCTS, PNN_STATIC_MAX_EDGES = 16384, 4096, 262144
PNN_STATIC_SCRATCH_BYTES, PNN_STATIC_EDGE_OVERFLOW = 6 * 1024 * 1024, 1
PNN_IMAGES_MINIMUM, PNN_IMAGES_ALL = 0, 1
PRECISIONS = {"bf16": PNN_BF16, "fp32": PNN_FP32, "fp64": PNN_FP64}

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libpnn.so")
_lib = None


class PnnError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = f"{where}: {pnn_status_string(status)} ({status})"
        if status == -3:
            msg += f" — {pnn_last_cuda_error()}"
        super().__init__(msg)


class pnn_config(ctypes.Structure):
    _fields_ = [("F", ctypes.c_int32), ("T", ctypes.c_int32), ("K", ctypes.c_int32), ("H", ctypes.c_int32),
                ("Zmax", ctypes.c_int32), ("cutoff", ctypes.c_double), ("norm_eps", ctypes.c_double),
                ("prec", ctypes.c_int32), ("rbf", ctypes.c_int32), ("pbc_images", ctypes.c_int32),
                ("max_neighbors", ctypes.c_int32), ("n_global", ctypes.c_int32), ("head_type", ctypes.c_int32),
                ("head_d1", ctypes.c_int32), ("head_d2", ctypes.c_int32), ("backbone", ctypes.c_int32)]


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Loads libpnn.so (built in-tree by paper_2604_15380_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} not found: build it with `python -m paper_2604_15380_b200.build` "
                              "(the CUDA library is the product; there is no fallback)")
        L = ctypes.CDLL(_LIB_PATH)
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
        L.pnn_status_string.restype = ctypes.c_char_p
        L.pnn_status_string.argtypes = [i32]
        L.pnn_last_cuda_error.restype = ctypes.c_char_p
        L.pnn_last_cuda_error.argtypes = []
        L.pnn_weights_count.argtypes = [ctypes.POINTER(pnn_config), ctypes.POINTER(i64)]
        L.pnn_model_create.argtypes = [ctypes.POINTER(pnn_config), vp, i64, ctypes.POINTER(vp)]
        L.pnn_model_destroy.argtypes = [vp]
        L.pnn_model_destroy.restype = None
        L.pnn_workspace_create.argtypes = [vp, i64, i64, i64, i32, ctypes.POINTER(vp)]
        L.pnn_workspace_destroy.argtypes = [vp]
        L.pnn_workspace_destroy.restype = None
        L.pnn_workspace_bytes.argtypes = [vp]
        L.pnn_workspace_bytes.restype = i64
        L.pnn_workspace_edge_tape_bytes.argtypes = [vp]
        L.pnn_workspace_edge_tape_bytes.restype = i64
        L.pnn_build_graph.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
        L.pnn_graph_view.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp),
                                     ctypes.POINTER(i64)]
        L.pnn_graph_copy.argtypes = [vp, vp, vp, vp]
        L.pnn_build_graph_static.argtypes = [i64, i64, vp, vp, vp, vp, ctypes.c_double, ctypes.c_int32, i64, vp, vp, vp, vp, vp]
        L.pnn_eval.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, i32, vp, vp, vp]
        L.pnn_set_globals.argtypes = [vp, i64, vp]
        L.pnn_eval_replay.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp]
        L.pnn_eval_blended.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, ctypes.c_double, i32, vp, vp, vp]
        L.pnn_eval_host.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp]
        L.pnn_branch_mlp_create.argtypes = [i32, vp, vp, i64, i32, ctypes.POINTER(vp)]
        L.pnn_branch_mlp_destroy.argtypes = [vp]
        L.pnn_branch_mlp_destroy.restype = None
        L.pnn_branch_weights.argtypes = [vp, vp, i64, i64, vp, vp, vp, vp]
        L.pnn_stream_create.argtypes = [vp, i64, i64, i64, i32, i32, ctypes.POINTER(vp)]
        L.pnn_stream_destroy.argtypes = [vp]
        L.pnn_stream_destroy.restype = None
        L.pnn_stream_submit.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, vp, vp]
        L.pnn_stream_wait.argtypes = [vp]
        L.pnn_stream_drain.argtypes = [vp]
        L.pnn_stream_launch_count.argtypes = [vp]
        L.pnn_stream_launch_count.restype = i64
        L.pnn_stream_bytes.argtypes = [vp]
        L.pnn_stream_bytes.restype = i64
        L.pnn_check_async_errors.argtypes = [vp]
        L.pnn_profile_enable.argtypes = [vp, i32]
        L.pnn_profile_read.argtypes = [vp, i32, vp, vp, vp, ctypes.POINTER(i32)]
        L.pnn_gemm_bf16.argtypes = [i64, i32, i32, vp, i64, vp, i64, vp, i32, vp, i64, vp, i64, vp]
        L.pnn_measure_alu_peak.argtypes = [i32, ctypes.POINTER(ctypes.c_double), vp]
        L.pnn_measure_l2_peak.argtypes = [ctypes.POINTER(ctypes.c_double), vp]
        L.pnn_launch_count.argtypes = [vp]
        L.pnn_launch_count.restype = i64
        _lib = L
    return _lib


def _check(st: int, where: str):
    if st != PNN_OK:
        raise PnnError(st, where)


_NP_DTYPES = {"i32": np.int32, "f64": np.float64, "f32": np.float32, "u8": np.uint8, "i8": np.int8}


def _ptr(x, dtype: Optional[str] = None, device: Optional[bool] = None, contiguous: bool = True) -> Optional[int]:
    """int / None pass through; numpy arrays give their host address; torch tensors their data_ptr().
    dtype ("i32", "f64", "f32", "u8", "i8", "bf16") and device (True: CUDA, False: host) are checked when given: the C ABI
    takes untyped pointers, so a wrong element type or a host pointer where a device one is expected would be misread."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        if dtype is not None and dtype != "bf16" and x.dtype != _NP_DTYPES[dtype]:
            raise TypeError(f"expected a {dtype} array, got {x.dtype}")
        if device:
            raise TypeError("expected a CUDA tensor, got a host array")
        return x.ctypes.data
    if contiguous and not x.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None:
        import torch
        want = {"i32": torch.int32, "f64": torch.float64, "f32": torch.float32, "u8": torch.uint8, "i8": torch.int8,
                "bf16": torch.bfloat16}[dtype]
        if x.dtype != want:
            raise TypeError(f"expected a {dtype} tensor, got {x.dtype}")
    if device is not None and bool(x.is_cuda) != device:
        raise TypeError("expected a CUDA tensor" if device else "expected a host tensor")
    return x.data_ptr()


def pnn_status_string(status: int) -> str:
    return lib().pnn_status_string(status).decode()


def pnn_last_cuda_error() -> str:
    return lib().pnn_last_cuda_error().decode()


def pnn_weights_count(cfg: pnn_config) -> int:
    n = ctypes.c_int64(0)
    _check(lib().pnn_weights_count(ctypes.byref(cfg), ctypes.byref(n)), "pnn_weights_count")
    return n.value


def pnn_model_create(cfg: pnn_config, weights_host: np.ndarray) -> int:
    w = np.ascontiguousarray(weights_host, np.float64)
    out = ctypes.c_void_p()
    _check(lib().pnn_model_create(ctypes.byref(cfg), w.ctypes.data, w.size, ctypes.byref(out)), "pnn_model_create")
    return out.value


def pnn_model_destroy(model: int) -> None:
    lib().pnn_model_destroy(model)


PNN_WS_FORCES, PNN_WS_NO_EDGE_TAPE = 1, 2


def pnn_workspace_create(model: int, max_atoms: int, max_edges: int, max_structs: int, want_forces) -> int:
    """want_forces: bool, or the PNN_WS_* flags of include/pnn.h."""
    out = ctypes.c_void_p()
    flags = int(want_forces) if not isinstance(want_forces, bool) else int(want_forces)
    _check(lib().pnn_workspace_create(model, max_atoms, max_edges, max_structs, flags, ctypes.byref(out)),
           "pnn_workspace_create")
    return out.value


def pnn_workspace_edge_tape_bytes(ws: int) -> int:
    return lib().pnn_workspace_edge_tape_bytes(ws)


def pnn_workspace_destroy(ws: int) -> None:
    lib().pnn_workspace_destroy(ws)


def pnn_workspace_bytes(ws: int) -> int:
    return lib().pnn_workspace_bytes(ws)


def pnn_build_graph(ws: int, n_atoms: int, n_structs: int, pos, struct_ptr, cell=None, pbc=None, stream=None):
    _check(lib().pnn_build_graph(ws, n_atoms, n_structs, _ptr(pos, "f64", True), _ptr(struct_ptr, "i32", True),
                                 _ptr(cell, "f64", True), _ptr(pbc, "u8", True), stream), "pnn_build_graph")


def pnn_graph_view(ws: int):
    """(rowptr_ptr, col_ptr, shift_ptr, n_edges); synchronises the build stream."""
    r, c, s = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_void_p()
    n = ctypes.c_int64(0)
    _check(lib().pnn_graph_view(ws, ctypes.byref(r), ctypes.byref(c), ctypes.byref(s), ctypes.byref(n)),
           "pnn_graph_view")
    return r.value, c.value, s.value, n.value


def pnn_graph_copy(ws: int, rowptr=None, col=None, shift=None):
    _check(lib().pnn_graph_copy(ws, _ptr(rowptr, "i32"), _ptr(col, "i32"), _ptr(shift, "i8")), "pnn_graph_copy")


def pnn_build_graph_static(n_atoms: int, n_structs: int, pos, struct_ptr, cell, pbc, cutoff: float, pbc_images: int,
                           max_edges: int, rowptr, col, shift, flags=None, stream=None) -> None:
    """The radius graph into caller-owned DEVICE buffers with no allocation inside the library (include/pnn.h: scratch in a
    static device array of PNN_STATIC_SCRATCH_BYTES; sizes beyond PNN_STATIC_MAX_* raise PnnError(-2) naming the limit)."""
    st = lib().pnn_build_graph_static(n_atoms, n_structs, _ptr(pos, "f64", True), _ptr(struct_ptr, "i32", True),
                                      _ptr(cell, "f64", True), _ptr(pbc, "u8", True), float(cutoff), int(pbc_images),
                                      max_edges, _ptr(rowptr, "i32", True), _ptr(col, "i32", True),
                                      _ptr(shift, "i8", True), _ptr(flags, "i32", True), stream)
    if st == -2:
        raise PnnError(st, "pnn_build_graph_static: " + pnn_last_cuda_error())
    _check(st, "pnn_build_graph_static")


def pnn_eval(model: int, ws: int, n_atoms: int, n_structs: int, Z, pos, struct_ptr, head, flags: int, energy,
             forces=None, stream=None):
    _check(lib().pnn_eval(model, ws, n_atoms, n_structs, _ptr(Z, "i32", True), _ptr(pos, "f64", True),
                          _ptr(struct_ptr, "i32", True), _ptr(head, "i32", True), flags, _ptr(energy, None, True),
                          _ptr(forces, None, True), stream), "pnn_eval")


def pnn_eval_replay(model: int, ws: int, n_atoms: int, n_structs: int, Z, pos, struct_ptr, head, cell, pbc, flags: int,
                    energy, forces=None, stream=None):
    """pnn_build_graph + pnn_eval as one replayed CUDA graph (include/pnn.h): same buffers, positions updated in place."""
    _check(lib().pnn_eval_replay(model, ws, n_atoms, n_structs, _ptr(Z, "i32", True), _ptr(pos, "f64", True),
                                 _ptr(struct_ptr, "i32", True), _ptr(head, "i32", True), _ptr(cell, "f64", True),
                                 _ptr(pbc, "u8", True), flags, _ptr(energy, None, True), _ptr(forces, None, True), stream),
           "pnn_eval_replay")


def pnn_set_globals(ws: int, n_structs: int, glob) -> None:
    _check(lib().pnn_set_globals(ws, n_structs, _ptr(glob, "f64", True)), "pnn_set_globals")


def pnn_eval_blended(model: int, ws: int, n_atoms: int, n_structs: int, Z, pos, struct_ptr, head_weights,
                     skip_below: float, flags: int, energy, forces=None, stream=None):
    _check(lib().pnn_eval_blended(model, ws, n_atoms, n_structs, _ptr(Z, "i32", True), _ptr(pos, "f64", True),
                                  _ptr(struct_ptr, "i32", True), _ptr(head_weights, None, True), float(skip_below), flags,
                                  _ptr(energy, None, True), _ptr(forces, None, True), stream), "pnn_eval_blended")


def pnn_branch_mlp_create(widths, params_host: np.ndarray, prec: int) -> int:
    w = np.ascontiguousarray(widths, dtype=np.int32)
    p = np.ascontiguousarray(params_host, dtype=np.float64)
    out = ctypes.c_void_p()
    _check(lib().pnn_branch_mlp_create(int(w.size) - 1, w.ctypes.data, p.ctypes.data, p.size, int(prec),
                                       ctypes.byref(out)), "pnn_branch_mlp_create")
    return out.value


def pnn_branch_mlp_destroy(b: int) -> None:
    lib().pnn_branch_mlp_destroy(b)


def pnn_branch_weights(b: int, ws: int, n_atoms: int, n_structs: int, Z, struct_ptr, head_weights, stream=None):
    _check(lib().pnn_branch_weights(b, ws, n_atoms, n_structs, _ptr(Z, "i32", True), _ptr(struct_ptr, "i32", True),
                                    _ptr(head_weights, None, True), stream), "pnn_branch_weights")


def pnn_eval_host(model: int, ws: int, n_atoms: int, n_structs: int, Z, pos, struct_ptr, head, cell, pbc,
                  flags: int, energy_host, forces_host=None, stream=None):
    _check(lib().pnn_eval_host(model, ws, n_atoms, n_structs, _ptr(Z, "i32", False), _ptr(pos, "f64", False),
                               _ptr(struct_ptr, "i32", False), _ptr(head, "i32", False), _ptr(cell, "f64", False),
                               _ptr(pbc, "u8", False), flags, _ptr(energy_host, None, False),
                               _ptr(forces_host, None, False), stream), "pnn_eval_host")


def pnn_stream_create(model: int, max_atoms: int, max_edges: int, max_structs: int, flags: int, depth: int = 2) -> int:
    out = ctypes.c_void_p()
    _check(lib().pnn_stream_create(model, max_atoms, max_edges, max_structs, flags, depth, ctypes.byref(out)),
           "pnn_stream_create")
    return out.value


def pnn_stream_destroy(s: int) -> None:
    lib().pnn_stream_destroy(s)


def pnn_stream_submit(s: int, n_atoms: int, n_structs: int, Z, pos, struct_ptr, head, cell, pbc, energy_host,
                      forces_host=None) -> None:
    """All HOST arrays (numpy or pinned torch CPU tensors); they must stay alive until the batch has been waited for."""
    _check(lib().pnn_stream_submit(s, n_atoms, n_structs, _ptr(Z, "i32", False), _ptr(pos, "f64", False),
                                   _ptr(struct_ptr, "i32", False), _ptr(head, "i32", False), _ptr(cell, "f64", False),
                                   _ptr(pbc, "u8", False), _ptr(energy_host, None, False), _ptr(forces_host, None, False)),
           "pnn_stream_submit")


def pnn_stream_wait(s: int) -> None:
    _check(lib().pnn_stream_wait(s), "pnn_stream_wait")


def pnn_stream_drain(s: int) -> None:
    _check(lib().pnn_stream_drain(s), "pnn_stream_drain")


def pnn_stream_launch_count(s: int) -> int:
    return lib().pnn_stream_launch_count(s)


def pnn_stream_bytes(s: int) -> int:
    return lib().pnn_stream_bytes(s)


def pnn_check_async_errors(ws: int) -> None:
    _check(lib().pnn_check_async_errors(ws), "pnn_check_async_errors")


def pnn_measure_alu_peak(prec: int, stream=None) -> float:
    """Measured TFLOP/s of the FMA pipe (packed FP32 or FP64 chains)."""
    out = ctypes.c_double()
    _check(lib().pnn_measure_alu_peak(int(prec), ctypes.byref(out), stream), "pnn_measure_alu_peak")
    return out.value


def pnn_measure_l2_peak(stream=None) -> float:
    """Measured GB/s of L2-resident reads (512-byte rows per warp)."""
    out = ctypes.c_double()
    _check(lib().pnn_measure_l2_peak(ctypes.byref(out), stream), "pnn_measure_l2_peak")
    return out.value


def pnn_launch_count(ws: int) -> int:
    return lib().pnn_launch_count(ws)


def pnn_profile_enable(ws: int, on: bool) -> None:
    _check(lib().pnn_profile_enable(ws, int(bool(on))), "pnn_profile_enable")


def pnn_profile_read(ws: int, max_entries: int = 32) -> dict:
    """{family: (total_ms, launches)} since the last read."""
    names = ctypes.create_string_buffer(32 * max_entries)
    ms = (ctypes.c_double * max_entries)()
    nl = (ctypes.c_int64 * max_entries)()
    n = ctypes.c_int(0)
    _check(lib().pnn_profile_read(ws, max_entries, ctypes.addressof(names), ctypes.addressof(ms),
                                  ctypes.addressof(nl), ctypes.byref(n)), "pnn_profile_read")
    return {names.raw[32 * q:32 * q + 32].split(b"\0")[0].decode(): (ms[q], nl[q]) for q in range(n.value)}


def pnn_gemm_bf16(M: int, N: int, K: int, A, lda: int, Wt, ldw: int, bias=None, act: int = 0, C=None, ldc: int = 0,
                  Cb=None, ldcb: int = 0, stream=None) -> None:
    sp = lambda t, dt: _ptr(t, dt, True, contiguous=False)   # row strides are explicit arguments here
    _check(lib().pnn_gemm_bf16(M, N, K, sp(A, "bf16"), lda, sp(Wt, "bf16"), ldw, sp(bias, "f32"), act, sp(C, "f32"), ldc,
                               sp(Cb, "bf16"), ldcb, stream), "pnn_gemm_bf16")


class PaiNN:
    """Model + workspace holder.  Marshals torch tensors / numpy arrays into the C ABI; no arithmetic here."""

    def __init__(self, F: int, T: int, K: int, H: int, weights: np.ndarray, *, precision: str = "fp32",
                 cutoff: float = 5.0, Zmax: int = 86, norm_eps: float = 1e-8, max_atoms: int, max_edges: int,
                 max_structs: int, forces: bool = True, rbf: str = "gaussian", pbc_images: str = "minimum",
                 edge_tape: bool = True, max_neighbors: int = 0, n_global: int = 0, head_type: str = "atomwise",
                 head_d1: int = 50, head_d2: int = 776, backbone: str = "painn"):
        self.cfg = pnn_config(F, T, K, H, Zmax, cutoff, norm_eps, PRECISIONS[precision],
                              {"gaussian": 0, "bessel": 1}[rbf], {"minimum": 0, "all": 1}[pbc_images], int(max_neighbors),
                              int(n_global), {"atomwise": 0, "pooled": 1}[head_type], int(head_d1), int(head_d2),
                              {"painn": 0, "schnet": 1}[backbone])
        self.precision = precision
        self.want_forces = bool(forces)
        self.model = pnn_model_create(self.cfg, weights)
        try:
            self.ws = pnn_workspace_create(self.model, max_atoms, max_edges, max_structs,
                                           (PNN_WS_FORCES if forces else 0) | (0 if edge_tape else PNN_WS_NO_EDGE_TAPE))
        except Exception:
            pnn_model_destroy(self.model)
            self.model = None
            raise
        self.max_atoms, self.max_edges, self.max_structs = max_atoms, max_edges, max_structs

    def close(self):
        if getattr(self, "branch_mlp", None):
            pnn_branch_mlp_destroy(self.branch_mlp)
            self.branch_mlp = None
        if getattr(self, "ws", None):
            pnn_workspace_destroy(self.ws)
            self.ws = None
        if getattr(self, "model", None):
            pnn_model_destroy(self.model)
            self.model = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def out_dtype(self):
        import torch
        return torch.float64 if self.precision == "fp64" else torch.float32

    @property
    def out_np_dtype(self):
        return np.float64 if self.precision == "fp64" else np.float32

    @staticmethod
    def _stream():
        import torch
        return torch.cuda.current_stream().cuda_stream

    def build_graph(self, pos, struct_ptr, cell=None, pbc=None):
        """pos [N,3] f64, struct_ptr [S+1] i32, cell [S,3,3] f64, pbc [S,3] u8: CUDA tensors."""
        N, S = int(pos.shape[0]), int(struct_ptr.shape[0]) - 1
        pnn_build_graph(self.ws, N, S, pos, struct_ptr, cell, pbc, self._stream())

    def graph(self):
        """Host copies (numpy) of rowptr [N+1], col [E], shift [E,3]."""
        _, _, _, E = pnn_graph_view(self.ws)
        N = self._last_N
        rowptr = np.zeros(N + 1, np.int32)
        col = np.zeros(E, np.int32)
        shift = np.zeros((E, 3), np.int8)
        pnn_graph_copy(self.ws, rowptr, col, shift)
        return rowptr, col, shift

    def eval(self, Z, pos, struct_ptr, head, cell=None, pbc=None, forces: Optional[bool] = None, build: bool = True,
             globals_=None):
        """CUDA tensors in, CUDA tensors out: (energy [S], forces [N,3] or None).  globals_: [S, n_global] f64 CUDA tensor
        of global attributes (charge, spin), or None."""
        import torch
        forces = self.want_forces if forces is None else forces
        N, S = int(Z.shape[0]), int(head.shape[0])
        self._last_N = N
        if self.cfg.n_global > 0:
            pnn_set_globals(self.ws, S, globals_)
        if build:
            self.build_graph(pos, struct_ptr, cell, pbc)
        energy = torch.empty(S, dtype=self.out_dtype, device=pos.device)
        frc = torch.empty((N, 3), dtype=self.out_dtype, device=pos.device) if forces else None
        flags = PNN_ENERGY | (PNN_FORCES if forces else 0)
        pnn_eval(self.model, self.ws, N, S, Z, pos, struct_ptr, head, flags, energy, frc, self._stream())
        return energy, frc

    def eval_replay(self, Z, pos, struct_ptr, head, energy, forces=None, cell=None, pbc=None):
        """Graph build + evaluation as one replayed CUDA graph (pnn_eval_replay): the caller owns ALL buffers, inputs and
        outputs (CUDA tensors), keeps them alive and updates `pos` in place between calls; forces=None: energy only."""
        N, S = int(Z.shape[0]), int(head.shape[0])
        self._last_N = N
        flags = PNN_ENERGY | (PNN_FORCES if forces is not None else 0)
        pnn_eval_replay(self.model, self.ws, N, S, Z, pos, struct_ptr, head, cell, pbc, flags, energy, forces,
                        self._stream())
        return energy, forces

    def eval_blended(self, Z, pos, struct_ptr, head_weights, cell=None, pbc=None, forces: Optional[bool] = None,
                     skip_below: float = 0.0, build: bool = True):
        """Blended multi-head evaluation: head_weights [S,H] CUDA tensor in the model's output dtype."""
        import torch
        forces = self.want_forces if forces is None else forces
        N, S = int(Z.shape[0]), int(head_weights.shape[0])
        self._last_N = N
        if build:
            self.build_graph(pos, struct_ptr, cell, pbc)
        energy = torch.empty(S, dtype=self.out_dtype, device=pos.device)
        frc = torch.empty((N, 3), dtype=self.out_dtype, device=pos.device) if forces else None
        flags = PNN_ENERGY | (PNN_FORCES if forces else 0)
        pnn_eval_blended(self.model, self.ws, N, S, Z, pos, struct_ptr, head_weights, skip_below, flags, energy, frc,
                         self._stream())
        return energy, frc

    def set_branch_mlp(self, widths, params: np.ndarray):
        """Uploads the composition -> softmax router; widths[-1] must equal H."""
        if int(widths[-1]) != self.cfg.H:
            raise ValueError("the router's last width must equal the number of heads")
        if getattr(self, "branch_mlp", None):
            pnn_branch_mlp_destroy(self.branch_mlp)
        self.branch_mlp = pnn_branch_mlp_create(widths, params, self.cfg.prec)

    def branch_weights(self, Z, struct_ptr):
        """[S,H] CUDA tensor of branch weights in the model's output dtype (the input of eval_blended)."""
        import torch
        if not getattr(self, "branch_mlp", None):
            raise RuntimeError("set_branch_mlp first")
        N, S = int(Z.shape[0]), int(struct_ptr.shape[0]) - 1
        hw = torch.empty((S, self.cfg.H), dtype=self.out_dtype, device=Z.device)
        pnn_branch_weights(self.branch_mlp, self.ws, N, S, Z, struct_ptr, hw, self._stream())
        return hw

    def eval_host(self, Z, pos, struct_ptr, head, cell=None, pbc=None, forces: Optional[bool] = None,
                  energy_out=None, forces_out=None):
        """Host numpy arrays (or pinned torch CPU tensors) in and out; H2D/D2H copies happen inside the library."""
        forces = self.want_forces if forces is None else forces
        N, S = int(Z.shape[0]), int(head.shape[0])
        self._last_N = N
        if energy_out is None:
            energy_out = np.empty(S, self.out_np_dtype)
        if forces and forces_out is None:
            forces_out = np.empty((N, 3), self.out_np_dtype)
        flags = PNN_ENERGY | (PNN_FORCES if forces else 0)
        pnn_eval_host(self.model, self.ws, N, S, Z, pos, struct_ptr, head, cell, pbc, flags, energy_out,
                      forces_out if forces else None, self._stream())
        return energy_out, (forces_out if forces else None)

    def check(self):
        pnn_check_async_errors(self.ws)

    @property
    def launches(self) -> int:
        return pnn_launch_count(self.ws)
