"""ctypes binding of include/mlp.h (same names, argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_NAME = "libpainn_b200.so"

EXPORTED_SYMBOLS = [
    "mlp_create", "mlp_compute", "mlp_compute_host", "mlp_destroy", "mlp_get_neighbors", "mlp_get_layer_state",
    "mlp_get_stats", "mlp_get_stage_ms", "mlp_set_option", "mlp_last_error", "mlp_version", "mlp_debug_gemm",
    "mlp_measure_row_gather", "mlp_row_offsets_static", "mlp_debug_row_offsets",
]

ERR_NAMES = {0: "MLP_OK", 1: "MLP_ERR_ARG", 2: "MLP_ERR_WEIGHTS", 3: "MLP_ERR_BOX_TOO_SMALL", 4: "MLP_ERR_TYPE_RANGE",
             5: "MLP_ERR_NOMEM", 6: "MLP_ERR_CUDA", 7: "MLP_ERR_NONFINITE"}


class MLPError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__(f"{ERR_NAMES.get(code, code)}: {msg}")


class _Stats(C.Structure):
    _fields_ = [("n_atoms", C.c_longlong), ("n_edges", C.c_longlong), ("atom_capacity", C.c_longlong),
                ("edge_capacity", C.c_longlong), ("n_cells", C.c_longlong * 3), ("n_regrow", C.c_longlong),
                ("n_calls", C.c_longlong), ("n_launches", C.c_longlong), ("device_bytes", C.c_longlong),
                ("n_list_rebuilds", C.c_longlong), ("n_list_reuses", C.c_longlong), ("n_graph_replays", C.c_longlong),
                ("n_reached", C.c_longlong)]


_lib = None


def lib_path() -> str:
    return os.path.join(_HERE, _LIB_NAME)


def load_library(build_if_missing: bool = True):
    """Load libpainn_b200.so (building it with nvcc first if it is missing or stale).  Raises if unavailable --
    there is deliberately no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if build_if_missing:
        from .build import build
        path = build()
    if not os.path.exists(path):
        raise ImportError(f"{path} not built; run `python -m paper_2506_04055_b200.build`")
    lib = C.CDLL(path)
    vp, ll, i32, dbl = C.c_void_p, C.c_longlong, C.c_int, C.c_double
    lib.mlp_create.argtypes = [vp, C.c_size_t, i32, dbl, ll, C.POINTER(vp)]
    lib.mlp_compute.argtypes = [vp, vp, vp, C.POINTER(dbl), ll, ll, vp, vp, vp, vp, vp]
    lib.mlp_compute_host.argtypes = [vp, vp, vp, C.POINTER(dbl), ll, ll, vp, vp, vp, vp]
    lib.mlp_destroy.argtypes = [vp]
    lib.mlp_destroy.restype = None
    lib.mlp_get_neighbors.argtypes = [vp, C.POINTER(ll), vp, vp, vp]
    lib.mlp_get_layer_state.argtypes = [vp, i32, vp]
    lib.mlp_get_stats.argtypes = [vp, C.POINTER(_Stats)]
    lib.mlp_get_stage_ms.argtypes = [vp, i32, C.POINTER(C.c_char_p), C.POINTER(C.c_float)]
    lib.mlp_set_option.argtypes = [vp, C.c_char_p, ll]
    lib.mlp_debug_gemm.argtypes = [vp, vp, vp, vp, ll, i32, i32, i32, i32, C.POINTER(i32)]
    lib.mlp_debug_gemm.restype = i32
    lib.mlp_measure_row_gather.argtypes = [ll, i32, C.POINTER(dbl)]
    lib.mlp_measure_row_gather.restype = i32
    for n in ("mlp_row_offsets_static", "mlp_debug_row_offsets"):
        getattr(lib, n).argtypes = [vp, vp, ll, vp, vp]
        getattr(lib, n).restype = i32
    lib.mlp_last_error.argtypes = [vp]
    lib.mlp_last_error.restype = C.c_char_p
    lib.mlp_version.restype = C.c_char_p
    for n in ("mlp_create", "mlp_compute", "mlp_compute_host", "mlp_get_neighbors", "mlp_get_layer_state",
              "mlp_get_stats", "mlp_get_stage_ms", "mlp_set_option"):
        getattr(lib, n).restype = i32
    _lib = lib
    return lib


def version() -> str:
    return load_library().mlp_version().decode()


def measure_row_gather(table_bytes: int = 2 << 30, window: int = 400) -> float:
    """GB/s the device sustains for the 512-byte row gather of the edge kernels (mlp_measure_row_gather)."""
    lib = load_library()
    out = C.c_double(0.0)
    rc = lib.mlp_measure_row_gather(int(table_bytes), int(window), C.byref(out))
    if rc != 0:
        raise MLPError(rc, "mlp_measure_row_gather")
    return out.value


ROW_OFFSETS_STATIC_MAX = 67108864      # mlp.h: MLP_ROW_OFFSETS_STATIC_MAX


def row_offsets(counts, static=True, stream=None):
    """Exclusive scan of a cuda int32 tensor of row counts -> (offsets[n + 1] int32, total int64 tensor).
    static=True: mlp_row_offsets_static (allocates nothing inside the library; the outputs are torch tensors made here);
    static=False: mlp_debug_row_offsets (the scan kernels of mlp_compute with a cudaMalloc'ed block buffer)."""
    import torch
    lib = load_library()
    assert counts.is_cuda and counts.dtype == torch.int32 and counts.is_contiguous()
    n = counts.numel()
    offsets = torch.empty(n + 1, dtype=torch.int32, device=counts.device)
    total = torch.empty(1, dtype=torch.int64, device=counts.device)
    return row_offsets_into(counts, offsets, total, static=static, stream=stream)


def row_offsets_into(counts, offsets, total, static=True, stream=None, n=None):
    """Same with caller-provided outputs (no torch allocation either).  `total` may be None for the static entry."""
    import torch
    lib = load_library()
    n = counts.numel() if n is None else int(n)
    st = torch.cuda.current_stream(counts.device).cuda_stream if stream is None else int(stream)
    fn = lib.mlp_row_offsets_static if static else lib.mlp_debug_row_offsets
    rc = fn(counts.data_ptr() if counts.numel() else None, offsets.data_ptr(), n,
            total.data_ptr() if total is not None else None, st)
    if rc != 0:
        raise MLPError(rc, fn.__name__)
    return offsets, total


def debug_gemm(A, W, bias=None, C_out=None, accumulate=False, path=0):
    """C (+)= A @ W.T + bias through the library's linear-layer kernel.  A, C_out: cuda float32 tensors; W, bias:
    numpy float32 (host).  Returns (C, used_tensor_cores)."""
    import torch
    lib = load_library()
    M, K = A.shape
    N = W.shape[0]
    W = np.ascontiguousarray(W, np.float32)
    assert W.shape == (N, K) and A.is_cuda and A.dtype == torch.float32 and A.is_contiguous()
    if C_out is None:
        C_out = torch.zeros((M, N), dtype=torch.float32, device=A.device)
    b = None if bias is None else np.ascontiguousarray(bias, np.float32)
    used = C.c_int(0)
    torch.cuda.synchronize()
    rc = lib.mlp_debug_gemm(A.data_ptr(), W.ctypes.data, None if b is None else b.ctypes.data, C_out.data_ptr(), M, N, K,
                            int(accumulate), int(path), C.byref(used))
    if rc != 0:
        raise MLPError(rc, "mlp_debug_gemm")
    return C_out, bool(used.value)


class Model:
    """mlp_create / mlp_compute / mlp_destroy with torch tensors (device) or numpy arrays (host)."""

    def __init__(self, weights: bytes, n_species: int, cutoff: float, capacity: int):
        self._lib = load_library()
        self._h = C.c_void_p()
        self._blob = bytes(weights)
        rc = self._lib.mlp_create(self._blob, len(self._blob), n_species, float(cutoff), int(capacity),
                                  C.byref(self._h))
        if rc != 0:
            self._h = C.c_void_p()
            raise MLPError(rc, "mlp_create")
        import struct
        self.F, self.K, self.T = struct.unpack_from("<3I", self._blob, 12)

    # -- helpers
    def _check(self, rc):
        if rc != 0:
            raise MLPError(rc, self._lib.mlp_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.mlp_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the hot path, device buffers (torch CUDA tensors)
    def compute(self, pos, types, box, n_local=None, n_ghost=0, ghost_owner=None, out=None, stream=None):
        """pos: cuda float64 [N,3]; types: cuda int32 [N]; box: 3 floats (host).  Returns (energy[1], forces[N,3],
        virial[6]) as cuda float64 tensors (asynchronous on the current / given torch stream)."""
        import torch
        if not (pos.is_cuda and types.is_cuda):
            raise MLPError(1, "compute() needs CUDA tensors; use compute_host() for host arrays")
        assert pos.dtype == torch.float64 and types.dtype == torch.int32 and pos.is_contiguous() and types.is_contiguous()
        N = pos.shape[0]
        n_local = N - n_ghost if n_local is None else n_local
        if out is None:
            out = (torch.empty(1, dtype=torch.float64, device=pos.device),
                   torch.empty((N, 3), dtype=torch.float64, device=pos.device),
                   torch.empty(6, dtype=torch.float64, device=pos.device))
        e, f, w = out
        boxc = (C.c_double * 3)(*[float(x) for x in box])
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        go = None
        if ghost_owner is not None:
            assert ghost_owner.is_cuda and ghost_owner.dtype == torch.int32 and ghost_owner.is_contiguous()
            go = ghost_owner.data_ptr()
        self._check(self._lib.mlp_compute(self._h, pos.data_ptr() if N else None, types.data_ptr() if N else None, boxc,
                                          int(n_local), int(n_ghost), go, e.data_ptr(),
                                          f.data_ptr() if N else None, w.data_ptr(), st.cuda_stream))
        return e, f, w

    # -- the same call with host buffers (numpy); copies happen inside the library
    def compute_host(self, pos, types, box, n_local=None, n_ghost=0, ghost_owner=None, out=None):
        pos = np.ascontiguousarray(pos, np.float64)
        types = np.ascontiguousarray(types, np.int32)
        N = pos.shape[0]
        n_local = N - n_ghost if n_local is None else n_local
        if out is None:
            out = (np.zeros(1), np.zeros((N, 3)), np.zeros(6))
        e, f, w = out
        boxc = (C.c_double * 3)(*[float(x) for x in box])
        go = None
        if ghost_owner is not None:
            ghost_owner = np.ascontiguousarray(ghost_owner, np.int32)
            go = ghost_owner.ctypes.data
        self._check(self._lib.mlp_compute_host(self._h, pos.ctypes.data, types.ctypes.data, boxc, int(n_local),
                                               int(n_ghost), go, e.ctypes.data, f.ctypes.data, w.ctypes.data))
        return e, f, w

    # -- debug / test exports
    def neighbors(self):
        """(i, j, image[E,3]) of the last compute, caller indices, sorted by (i, j, image)."""
        n = C.c_longlong(0)
        self._check(self._lib.mlp_get_neighbors(self._h, C.byref(n), None, None, None))
        E = n.value
        i = np.empty(max(E, 1), np.int32); j = np.empty(max(E, 1), np.int32); im = np.empty((max(E, 1), 3), np.int8)
        self._check(self._lib.mlp_get_neighbors(self._h, C.byref(n), i.ctypes.data, j.ctypes.data, im.ctypes.data))
        i, j, im = i[:E], j[:E], im[:E]
        order = np.lexsort((im[:, 2], im[:, 1], im[:, 0], j, i))
        return i[order], j[order], im[order]

    def layer_state(self, t: int, n_atoms: int):
        out = np.empty((n_atoms, 4 * self.F), np.float32)
        self._check(self._lib.mlp_get_layer_state(self._h, int(t), out.ctypes.data))
        return out

    def stats(self) -> dict:
        s = _Stats()
        self._check(self._lib.mlp_get_stats(self._h, C.byref(s)))
        d = {k: getattr(s, k) for k, _ in _Stats._fields_ if k != "n_cells"}
        d["n_cells"] = tuple(s.n_cells)
        return d

    def set_option(self, name: str, value: int):
        self._check(self._lib.mlp_set_option(self._h, name.encode(), int(value)))

    def stage_ms(self) -> dict:
        names = (C.c_char_p * 16)()
        ms = (C.c_float * 16)()
        n = self._lib.mlp_get_stage_ms(self._h, 16, names, ms)
        if n < 0:
            raise MLPError(-n, "mlp_get_stage_ms")
        return {names[k].decode(): float(ms[k]) for k in range(n)}
