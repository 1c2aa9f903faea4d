"""paper_2607_06604_b200 -- thin Python binding of the C-ABI CUDA library ``libgramsci.so``.

Argument marshalling only: every step of the path (graph build, 2/3/4-point enumeration, parity split,
fold, out-of-core tiling) runs in the CUDA kernels behind ``include/gramsci.h``.  PyTorch is used for
device memory and streams.  There is no CPU fallback: importing works without a GPU (so that the
symbol table can be checked), but every compute call fails loudly when the library or a CUDA device
is missing.

Functions mirror the ABI names: :func:`gramsci_build_graph` -> :class:`Graph` with methods
``pcf2 / pcf3 / pcf4 / pcf4_parity`` (= ``gramsci_2pcf`` ...), plus the host helpers
:func:`gramsci_num_configs`, :func:`gramsci_compact`, :func:`gramsci_zeta_disc`.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgramsci.so")

ABI_SYMBOLS = [
    "gramsci_build_graph", "gramsci_graph_info", "gramsci_export_csr", "gramsci_2pcf", "gramsci_3pcf",
    "gramsci_4pcf", "gramsci_4pcf_parity", "gramsci_num_configs", "gramsci_compact", "gramsci_zeta_disc",
    "gramsci_last_timing", "gramsci_work_counters", "gramsci_free_graph", "gramsci_last_error",
    "gramsci_export_labels", "gramsci_release_memory", "gramsci_3pcf_equilateral", "gramsci_slab_range",
    "gramsci_2pcf_noalloc",
]

NOALLOC_MAX_BINS = 128          # GRAMSCI_NOALLOC_MAX_BINS of include/gramsci.h (gramsci_2pcf_noalloc)

ALGO_DEFAULT, ALGO_MERGEPATH, ALGO_BSEARCH, ALGO_BITMAP = 0, 1, 2, 3
ALGO_TABLE_G1, ALGO_TABLE_G2, ALGO_TABLE_G4, ALGO_TABLE_G8 = 4, 5, 6, 7
ALGO_GATHER = 8

STATUS = {0: "GRAMSCI_OK", 1: "GRAMSCI_EINVAL", 2: "GRAMSCI_ERANGE", 3: "GRAMSCI_ENOMEM", 4: "GRAMSCI_ECUDA",
          5: "GRAMSCI_EOVERFLOW"}


class GramsciError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


_ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p)
_DEALLOC_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p)


class _Options(ctypes.Structure):
    _fields_ = [("stream", ctypes.c_void_p), ("device_mem_cap_bytes", ctypes.c_uint64),
                ("want_pixels", ctypes.c_int), ("relabel", ctypes.c_int), ("algo", ctypes.c_int),
                ("n_windows", ctypes.c_int), ("hub_stride", ctypes.c_int),
                ("shard_count", ctypes.c_int), ("shard_index", ctypes.c_int),
                ("slab_count", ctypes.c_int), ("slab_index", ctypes.c_int), ("reserved", ctypes.c_int),
                ("alloc", _ALLOC_FN), ("dealloc", _DEALLOC_FN), ("user", ctypes.c_void_p)]


def _torch_alloc(size, stream, user):
    """``gramsci_options.alloc`` hook: PyTorch's caching allocator (device memory belongs to torch)."""
    import torch
    try:
        return torch.cuda.caching_allocator_alloc(int(size), stream=int(stream or 0))
    except Exception:        # out of memory: the library reports GRAMSCI_ENOMEM
        return None


def _torch_dealloc(ptr, stream, user):
    import torch
    torch.cuda.caching_allocator_delete(int(ptr))


_TORCH_HOOKS = (_ALLOC_FN(_torch_alloc), _DEALLOC_FN(_torch_dealloc))     # kept alive for the life of the process


_lib = None


def load_library():
    """dlopen libgramsci.so (raises if it has not been built: ``python -m paper_2607_06604_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_06604_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, i64p = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int64)
    L.gramsci_build_graph.restype = ctypes.c_int
    L.gramsci_build_graph.argtypes = [vp, vp, ctypes.c_int64, ctypes.POINTER(ctypes.c_double), ctypes.c_double,
                                      ctypes.c_double, ctypes.c_int, ctypes.POINTER(_Options), ctypes.POINTER(vp)]
    L.gramsci_graph_info.restype = ctypes.c_int
    L.gramsci_graph_info.argtypes = [vp, i64p, i64p, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_uint64),
                                     ctypes.POINTER(ctypes.c_int32)]
    L.gramsci_export_csr.restype = ctypes.c_int
    L.gramsci_export_csr.argtypes = [vp] * 5
    for name, nargs in (("gramsci_2pcf", 3), ("gramsci_3pcf", 3), ("gramsci_3pcf_equilateral", 3), ("gramsci_4pcf", 3),
                        ("gramsci_4pcf_parity", 5)):
        f = getattr(L, name)
        f.restype = ctypes.c_int
        f.argtypes = [vp] * nargs
    L.gramsci_num_configs.restype = ctypes.c_int
    L.gramsci_num_configs.argtypes = [ctypes.c_int, ctypes.c_int, i64p]
    L.gramsci_compact.restype = ctypes.c_int
    L.gramsci_compact.argtypes = [ctypes.c_int, ctypes.c_int, vp, ctypes.c_int, vp, vp]
    L.gramsci_zeta_disc.restype = ctypes.c_int
    L.gramsci_zeta_disc.argtypes = [ctypes.c_int, vp, vp]
    L.gramsci_last_timing.restype = ctypes.c_int
    L.gramsci_last_timing.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    L.gramsci_work_counters.restype = ctypes.c_int
    L.gramsci_work_counters.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
    L.gramsci_free_graph.restype = None
    L.gramsci_free_graph.argtypes = [vp]
    L.gramsci_last_error.restype = ctypes.c_char_p
    L.gramsci_last_error.argtypes = []
    L.gramsci_export_labels.restype = ctypes.c_int
    L.gramsci_export_labels.argtypes = [vp, vp]
    L.gramsci_release_memory.restype = ctypes.c_int
    L.gramsci_release_memory.argtypes = []
    L.gramsci_2pcf_noalloc.restype = ctypes.c_int
    L.gramsci_2pcf_noalloc.argtypes = [vp] * 3
    L.gramsci_slab_range.restype = ctypes.c_int
    L.gramsci_slab_range.argtypes = [vp, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32)]
    _lib = L
    return L


def _check(code: int):
    if code != 0:
        raise GramsciError(code, load_library().gramsci_last_error().decode("utf-8", "replace"))


def _ptr(a) -> Optional[int]:
    """Raw address of a torch tensor (device or host) or a NumPy array (host); None passes NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.is_contiguous()
    return a.data_ptr()


def _is_torch(a) -> bool:
    return a is not None and not isinstance(a, np.ndarray)


def _current_stream_ptr() -> Optional[int]:
    import torch
    if not torch.cuda.is_available():
        return None
    return torch.cuda.current_stream().cuda_stream


class Graph:
    """Opaque handle of ``gramsci_graph`` (owned by the library, freed on garbage collection)."""

    def __init__(self, handle: int, nbins: int, device: bool):
        self._h = handle
        self.nbins = nbins
        self._device_outputs = device

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.gramsci_free_graph(h)

    free = __del__

    # -- info ---------------------------------------------------------------------------------------
    def info(self) -> dict:
        n, e = ctypes.c_int64(), ctypes.c_int64()
        mr, nw, cb = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_uint64()
        _check(load_library().gramsci_graph_info(self._h, ctypes.byref(n), ctypes.byref(e), ctypes.byref(mr),
                                                 ctypes.byref(cb), ctypes.byref(nw)))
        return dict(n_points=n.value, n_edges=e.value, max_row=mr.value, csr_bytes=cb.value, n_windows=nw.value)

    def slab_range(self):
        """``gramsci_slab_range``: the hubs this graph owns, [hub_lo, hub_hi) in internal labels."""
        lo, hi = ctypes.c_int32(), ctypes.c_int32()
        _check(load_library().gramsci_slab_range(self._h, ctypes.byref(lo), ctypes.byref(hi)))
        return lo.value, hi.value

    def timing(self, what: int) -> float:
        v = ctypes.c_double()
        _check(load_library().gramsci_last_timing(self._h, what, ctypes.byref(v)))
        return v.value

    def work_counters(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        _check(load_library().gramsci_work_counters(self._h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def export_csr(self, want_pix: bool = False):
        """CSR in caller labels as host NumPy arrays (ptr int64, idx int32, bin uint8[, pix uint8])."""
        inf = self.info()
        n, e = inf["n_points"], inf["n_edges"]
        ptr = np.zeros(n + 1, dtype=np.int64)
        idx = np.zeros(max(e, 1), dtype=np.int32)
        b = np.zeros(max(e, 1), dtype=np.uint8)
        p = np.zeros(max(e, 1), dtype=np.uint8) if want_pix else None
        _check(load_library().gramsci_export_csr(self._h, _ptr(ptr), _ptr(idx), _ptr(b), _ptr(p)))
        return (ptr, idx[:e], b[:e], p[:e]) if want_pix else (ptr, idx[:e], b[:e])

    def export_labels(self) -> np.ndarray:
        """``gramsci_export_labels``: caller index of every internal label (int32 [N], host)."""
        out = np.zeros(max(self.info()["n_points"], 1), dtype=np.int32)
        _check(load_library().gramsci_export_labels(self._h, _ptr(out)))
        return out[:self.info()["n_points"]]

    # -- outputs ------------------------------------------------------------------------------------
    def _out(self, n: int, dtype: str, host: bool):
        if host or not self._device_outputs:
            return np.zeros(n, dtype=dtype)
        import torch
        return torch.zeros(n, dtype=getattr(torch, dtype), device="cuda")

    @staticmethod
    def _np(a, view: Optional[str] = None):
        if a is None:
            return None
        if not isinstance(a, np.ndarray):
            a = a.cpu().numpy()
        return a.view(view) if view else a

    # -- queries (numpy results; pass host=True to let the library write straight into host memory) --
    def pcf2(self, weighted: bool = False, host: bool = False):
        nb = self.nbins
        c = self._out(nb, "int64", host)
        w = self._out(nb, "float64", host) if weighted else None
        _check(load_library().gramsci_2pcf(self._h, _ptr(c), _ptr(w)))
        return self._np(c), self._np(w)

    def pcf2_noalloc(self, counts=None, wsum=None):
        """``gramsci_2pcf_noalloc``: the 2pCF into the caller's CUDA tensors (int64 / float64 [nbins], either may be None)
        with no allocation inside the library.  The call only ENQUEUES work on the graph's stream; this wrapper then
        synchronises that stream (torch's current stream at build time) so that the tensors are complete on return."""
        import torch
        for t, dt in ((counts, torch.int64), (wsum, torch.float64)):
            assert t is None or (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() >= self.nbins)
        _check(load_library().gramsci_2pcf_noalloc(self._h, _ptr(counts), _ptr(wsum)))
        torch.cuda.synchronize()
        return counts, wsum

    def pcf3(self, counts: bool = True, weighted: bool = False, host: bool = False):
        nh = self.nbins ** 3
        c = self._out(nh, "int64", host) if counts else None
        w = self._out(nh, "float64", host) if weighted else None
        _check(load_library().gramsci_3pcf(self._h, _ptr(c), _ptr(w)))
        return self._np(c), self._np(w)

    def pcf3_equilateral(self, counts: bool = True, weighted: bool = False, host: bool = False):
        """``gramsci_3pcf_equilateral``: [nb] histograms of the triangles with all three edges in one bin."""
        c = self._out(self.nbins, "int64", host) if counts else None
        w = self._out(self.nbins, "float64", host) if weighted else None
        _check(load_library().gramsci_3pcf_equilateral(self._h, _ptr(c), _ptr(w)))
        return self._np(c), self._np(w)

    def pcf4(self, counts: bool = True, weighted: bool = False, host: bool = False):
        nh = self.nbins ** 6
        c = self._out(nh, "int64", host) if counts else None
        w = self._out(nh, "float64", host) if weighted else None
        _check(load_library().gramsci_4pcf(self._h, _ptr(c), _ptr(w)))
        return self._np(c), self._np(w)

    def pcf4_parity(self, counts: bool = True, weighted: bool = False, host: bool = False):
        nh = self.nbins ** 6
        ec = self._out(nh, "int64", host) if counts else None
        oc = self._out(nh, "int64", host) if counts else None
        ew = self._out(nh, "float64", host) if weighted else None
        ow = self._out(nh, "float64", host) if weighted else None
        _check(load_library().gramsci_4pcf_parity(self._h, _ptr(ec), _ptr(oc), _ptr(ew), _ptr(ow)))
        return self._np(ec), self._np(oc), self._np(ew), self._np(ow)


def gramsci_build_graph(points, weights=None, box: Optional[Sequence[float]] = None, r_min: float = 0.0,
                        r_max: float = 1.0, nbins: int = 1, *, want_pixels: bool = False, relabel: int = 0,
                        algo: int = 0, device_mem_cap_bytes: int = 0, n_windows: int = 0, hub_stride: int = 0,
                        shard_count: int = 0, shard_index: int = 0, slab_count: int = 0, slab_index: int = 0,
                        torch_allocator: bool = False) -> Graph:
    """``gramsci_build_graph`` (include/gramsci.h).  ``points`` [N,3] / ``weights`` [N] fp64: torch CUDA
    tensors (used in place), torch CPU tensors or NumPy arrays (the library stages host buffers itself)."""
    L = load_library()
    if isinstance(points, np.ndarray):
        points = np.ascontiguousarray(points, dtype=np.float64)
        n = points.shape[0]
    else:
        import torch
        assert points.dtype == torch.float64
        points = points.contiguous()
        n = points.shape[0]
    if weights is not None:
        if isinstance(weights, np.ndarray):
            weights = np.ascontiguousarray(weights, dtype=np.float64)
        else:
            weights = weights.contiguous()
    opt = _Options()
    opt.stream = _current_stream_ptr()
    opt.device_mem_cap_bytes = int(device_mem_cap_bytes)
    opt.want_pixels = int(bool(want_pixels))
    opt.relabel = int(relabel)
    opt.algo = int(algo)
    opt.n_windows = int(n_windows)
    opt.hub_stride = int(hub_stride)
    opt.shard_count = int(shard_count)
    opt.shard_index = int(shard_index)
    opt.slab_count = int(slab_count)
    opt.slab_index = int(slab_index)
    if torch_allocator:          # S:8(b): the graph and all scratch come from torch's caching allocator
        opt.alloc, opt.dealloc = _TORCH_HOOKS
    cbox = None
    if box is not None:
        cbox = (ctypes.c_double * 3)(*[float(v) for v in box])
    h = ctypes.c_void_p()
    code = L.gramsci_build_graph(_ptr(points), _ptr(weights), int(n),
                                 ctypes.cast(cbox, ctypes.POINTER(ctypes.c_double)) if cbox is not None else None,
                                 float(r_min), float(r_max), int(nbins), ctypes.byref(opt), ctypes.byref(h))
    _check(code)
    device = _is_torch(points) and points.is_cuda
    return Graph(h.value, int(nbins), device)


def gramsci_release_memory() -> None:
    _check(load_library().gramsci_release_memory())


def gramsci_num_configs(npoint: int, nbins: int) -> int:
    n = ctypes.c_int64()
    _check(load_library().gramsci_num_configs(npoint, nbins, ctypes.byref(n)))
    return n.value


def gramsci_compact(npoint: int, nbins: int, dense: np.ndarray):
    """(compact values [n_configs], config bins uint8 [n_configs, 3|6]) of a dense host histogram."""
    n = gramsci_num_configs(npoint, nbins)
    dense = np.ascontiguousarray(dense)
    assert dense.dtype.itemsize == 8
    out = np.zeros(n, dtype=dense.dtype)
    bins = np.zeros((n, 3 if npoint == 3 else 6), dtype=np.uint8)
    _check(load_library().gramsci_compact(npoint, nbins, _ptr(dense), 8, _ptr(out), _ptr(bins)))
    return out, bins


def gramsci_zeta_disc(xi: np.ndarray) -> np.ndarray:
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    out = np.zeros(xi.size ** 6, dtype=np.float64)
    _check(load_library().gramsci_zeta_disc(xi.size, _ptr(xi), _ptr(out)))
    return out
