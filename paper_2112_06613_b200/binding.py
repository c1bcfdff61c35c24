"""Thin ctypes binding of include/tcrnet.h: argument marshalling only.

Every step of the path (pack, schedule, distances, emission, sort, CSR, degrees) runs inside
libtcrnet_b200.so.  PyTorch is used for exactly three things: device memory (the library's
allocator callbacks are backed by ``torch.empty(..., device="cuda")``), the CUDA stream handle,
and zero-copy tensor views of the results.  There is no CPU fallback: if the shared library is
missing or no CUDA device is present, creation fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtcrnet_b200.so")

# status codes / options (mirrors of the enums in tcrnet.h)
OK, ERR_ARG, ERR_LENGTH, ERR_RESIDUE, ERR_LMAX, ERR_STATE, ERR_NOMEM, ERR_EDGE_OVERFLOW, ERR_CUDA = (
    0, -1, -2, -3, -4, -5, -6, -7, -8)
ERR_CAPACITY = -9
NOALLOC_MAX_ROWS = 1 << 21  # TCRNET_NOALLOC_MAX_ROWS
OPT_EARLY_EXIT, OPT_FIRST_CHECK, OPT_EDGE_CAPACITY, OPT_EDGE_LIMIT, OPT_COUNT_WORK, OPT_TEXT_CHUNK = 1, 2, 3, 4, 5, 6
OPT_PREFIX_TRIE, OPT_TRIE_CHUNK, OPT_N_QUERY, OPT_DEDUP, OPT_SEGMENT_JOIN, OPT_FAST_L1, OPT_TIMING = 7, 8, 9, 10, 11, 12, 13

EXPORTS = (
    "tcrnet_create", "tcrnet_destroy", "tcrnet_load", "tcrnet_load_sized", "tcrnet_load_device", "tcrnet_build",
    "tcrnet_csr", "tcrnet_row_ptr_noalloc",
    "tcrnet_degrees", "tcrnet_copy_csr", "tcrnet_set_option", "tcrnet_get_stats", "tcrnet_probe_int32",
    "tcrnet_last_cuda_error", "tcrnet_strerror", "tcrnet_version", "tcrnet_build_shard", "tcrnet_assemble",
    "tcrnet_edge_distances", "tcrnet_restrict", "tcrnet_degree_histogram", "tcrnet_neighbor_degree",
    "tcrnet_components", "tcrnet_percolation",
)


class tcrnet_allocator(C.Structure):
    ALLOC = C.CFUNCTYPE(C.c_void_p, C.c_void_p, C.c_size_t)
    FREE = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)
    _fields_ = [("alloc", ALLOC), ("free", FREE), ("user", C.c_void_p)]


class tcrnet_stats(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("total_len", C.c_int64), ("min_len", C.c_int32), ("max_len", C.c_int32),
        ("l_max", C.c_int32), ("first_check", C.c_int32), ("n_edges", C.c_int64), ("pairs_all", C.c_int64),
        ("pairs_kept", C.c_int64), ("cells_all", C.c_int64), ("cells_kept", C.c_int64),
        ("columns_kept", C.c_int64), ("lane_columns_exec", C.c_int64), ("lane_tests_exec", C.c_int64),
        ("lane_pairs_exec", C.c_int64), ("lane_prefix_tests_exec", C.c_int64), ("work_items", C.c_int64),
        ("work_items_trie", C.c_int64), ("trie_nodes", C.c_int64), ("distance_passes", C.c_int32),
        ("launches_load", C.c_int32), ("launches_build", C.c_int32), ("ms_load", C.c_float),
        ("ms_distance", C.c_float), ("ms_sort", C.c_float), ("ms_csr", C.c_float), ("ms_build", C.c_float),
        ("n_distinct", C.c_int64), ("ms_kernel", C.c_float), ("ms_index", C.c_float),
        ("lane_columns_live", C.c_int64), ("join_probes", C.c_int64), ("join_entries", C.c_int64),
        ("join_candidates", C.c_int64), ("work_items_join", C.c_int64), ("join_index_entries", C.c_int64),
        ("join_mode", C.c_int32), ("pad2_", C.c_int32), ("join_survivors", C.c_int64), ("join_diagonals", C.c_int64),
        ("join_verified_edges", C.c_int64),
        ("join_adapted_lengths", C.c_int32),
        ("pad3_", C.c_int32),
    ]


class TcrNetError(RuntimeError):
    def __init__(self, status: int, what: str):
        super().__init__(f"{what}: {strerror(status)} (status {status})")
        self.status = status


_lib = None


def load_library() -> C.CDLL:
    """dlopen the in-tree shared library (no GPU needed for this) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2112_06613_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i64p, i32p, u8p = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.POINTER(C.c_uint8)
    lib.tcrnet_create.restype = C.c_int
    lib.tcrnet_create.argtypes = [C.POINTER(vp), C.c_int, vp, C.POINTER(tcrnet_allocator)]
    lib.tcrnet_destroy.restype = None
    lib.tcrnet_destroy.argtypes = [vp]
    lib.tcrnet_load.restype = C.c_int
    lib.tcrnet_load.argtypes = [vp, u8p, i32p, C.c_int64]
    lib.tcrnet_load_sized.restype = C.c_int
    lib.tcrnet_load_sized.argtypes = [vp, u8p, C.c_int64, i32p, C.c_int64]
    lib.tcrnet_load_device.restype = C.c_int
    lib.tcrnet_load_device.argtypes = [vp, vp, vp, C.c_int64, C.c_int64]
    lib.tcrnet_build.restype = C.c_int
    lib.tcrnet_build.argtypes = [vp, C.c_int, i64p]
    lib.tcrnet_build_shard.restype = C.c_int
    lib.tcrnet_build_shard.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.POINTER(vp), i64p]
    lib.tcrnet_assemble.restype = C.c_int
    lib.tcrnet_assemble.argtypes = [vp, vp, C.c_int64, i64p]
    lib.tcrnet_edge_distances.restype = C.c_int
    lib.tcrnet_edge_distances.argtypes = [vp, C.POINTER(vp)]
    lib.tcrnet_restrict.restype = C.c_int
    lib.tcrnet_restrict.argtypes = [vp, C.c_int, i64p]
    lib.tcrnet_degree_histogram.restype = C.c_int
    lib.tcrnet_degree_histogram.argtypes = [vp, C.POINTER(vp), i32p]
    lib.tcrnet_neighbor_degree.restype = C.c_int
    lib.tcrnet_neighbor_degree.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    lib.tcrnet_components.restype = C.c_int
    lib.tcrnet_components.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), i64p, i64p]
    lib.tcrnet_percolation.restype = C.c_int
    lib.tcrnet_percolation.argtypes = [vp, i32p, i64p, C.c_int32, i64p, C.POINTER(C.c_double),
                                       C.POINTER(C.c_double), i64p]
    lib.tcrnet_csr.restype = C.c_int
    lib.tcrnet_csr.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    lib.tcrnet_row_ptr_noalloc.restype = C.c_int
    lib.tcrnet_row_ptr_noalloc.argtypes = [vp, C.c_int64, vp, vp, C.POINTER(C.c_int)]
    lib.tcrnet_degrees.restype = C.c_int
    lib.tcrnet_degrees.argtypes = [vp, C.POINTER(vp)]
    lib.tcrnet_copy_csr.restype = C.c_int
    lib.tcrnet_copy_csr.argtypes = [vp, i64p, i32p, i32p]
    lib.tcrnet_set_option.restype = C.c_int
    lib.tcrnet_set_option.argtypes = [vp, C.c_int, C.c_int64]
    lib.tcrnet_get_stats.restype = C.c_int
    lib.tcrnet_get_stats.argtypes = [vp, C.POINTER(tcrnet_stats)]
    lib.tcrnet_probe_int32.restype = C.c_int
    lib.tcrnet_probe_int32.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.tcrnet_last_cuda_error.restype = C.c_int
    lib.tcrnet_last_cuda_error.argtypes = [vp]
    lib.tcrnet_strerror.restype = C.c_char_p
    lib.tcrnet_strerror.argtypes = [C.c_int]
    lib.tcrnet_version.restype = C.c_int
    lib.tcrnet_version.argtypes = []
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load_library().tcrnet_strerror(int(status)).decode()


def version() -> int:
    return int(load_library().tcrnet_version())


def _check(status: int, what: str) -> None:
    if status != OK:
        raise TcrNetError(status, what)


class TcrNet:
    """One tcrnet_ctx.  Method names follow the C calls (tcrnet_load -> load, ...)."""

    def __init__(self, device: int = 0, stream=None):
        import torch  # device memory + stream only

        self._lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("tcrnet: no CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.device = torch.device("cuda", device)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._blocks: Dict[int, "torch.Tensor"] = {}
        self._staging: Dict[str, "torch.Tensor"] = {}  # page-locked host buffers of copy_csr(staged=True)

        def _alloc(_user, nbytes):
            try:
                with torch.cuda.stream(self._stream):
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            except Exception:  # torch.OutOfMemoryError and friends -> NULL -> TCRNET_ERR_NOMEM
                return None
            self._blocks[t.data_ptr()] = t
            return t.data_ptr()

        def _free(_user, ptr):
            self._blocks.pop(int(ptr) if ptr else 0, None)

        self._cb_alloc = tcrnet_allocator.ALLOC(_alloc)
        self._cb_free = tcrnet_allocator.FREE(_free)
        self._allocator = tcrnet_allocator(self._cb_alloc, self._cb_free, None)
        self._ctx = C.c_void_p()
        _check(self._lib.tcrnet_create(C.byref(self._ctx), device, C.c_void_p(self._stream.cuda_stream),
                                       C.byref(self._allocator)), "tcrnet_create")
        self.n = 0
        self.n_edges = 0

    # -- lifetime -------------------------------------------------------------------------
    def destroy(self) -> None:
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.tcrnet_destroy(self._ctx)
            self._ctx = C.c_void_p()
            self._blocks.clear()

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # -- the calls of tcrnet.h -------------------------------------------------------------
    def load(self, residues, lengths) -> None:
        """tcrnet_load_sized (host numpy arrays) or tcrnet_load_device (CUDA torch tensors)."""
        torch = self._torch
        if isinstance(residues, torch.Tensor):
            assert residues.is_cuda and lengths.is_cuda, "device load needs CUDA tensors"
            assert residues.dtype == torch.uint8 and lengths.dtype == torch.int32
            residues, lengths = residues.contiguous(), lengths.contiguous()
            n = int(lengths.numel())
            _check(self._lib.tcrnet_load_device(self._ctx, C.c_void_p(residues.data_ptr()),
                                                C.c_void_p(lengths.data_ptr()), n, int(residues.numel())),
                   "tcrnet_load_device")
        else:
            residues = np.ascontiguousarray(residues, dtype=np.uint8)
            lengths = np.ascontiguousarray(lengths, dtype=np.int32)
            n = int(lengths.size)
            # (tcrnet_load_sized checks sum(lengths) <= residues.size as it reads the lengths: no pass over them here)
            _check(self._lib.tcrnet_load_sized(self._ctx, residues.ctypes.data_as(C.POINTER(C.c_uint8)),
                                               int(residues.size), lengths.ctypes.data_as(C.POINTER(C.c_int32)), n),
                   "tcrnet_load")
        self.n = n
        self.n_edges = 0

    def build(self, l_max: int) -> int:
        e = C.c_int64(0)
        _check(self._lib.tcrnet_build(self._ctx, int(l_max), C.byref(e)), "tcrnet_build")
        self.n_edges = int(e.value)
        return self.n_edges

    def build_shard(self, l_max: int, shard: int, n_shards: int) -> "torch.Tensor":
        """tcrnet_build_shard: this shard's edge keys (i << 32) | j as an int64 CUDA tensor (a view of
        library memory, valid until the next build / assemble / restrict / load)."""
        torch = self._torch
        keys, e = C.c_void_p(), C.c_int64(0)
        _check(self._lib.tcrnet_build_shard(self._ctx, int(l_max), int(shard), int(n_shards), C.byref(keys),
                                            C.byref(e)), "tcrnet_build_shard")
        self.n_edges = 0
        if not e.value:
            return torch.empty(0, dtype=torch.int64, device=self.device)
        return self._view(keys.value, torch.int64, int(e.value))

    def assemble(self, keys: "torch.Tensor") -> int:
        """tcrnet_assemble: CSR + degrees from an int64 CUDA tensor of keys (i << 32) | j."""
        torch = self._torch
        assert keys.is_cuda and keys.dtype == torch.int64
        keys = keys.contiguous()
        e = C.c_int64(0)
        _check(self._lib.tcrnet_assemble(self._ctx, C.c_void_p(keys.data_ptr() if keys.numel() else 0),
                                         int(keys.numel()), C.byref(e)), "tcrnet_assemble")
        self.n_edges = int(e.value)
        return self.n_edges

    def edge_distances(self) -> "torch.Tensor":
        """tcrnet_edge_distances: uint8[E] aligned with col (a view of library memory)."""
        torch = self._torch
        d = C.c_void_p()
        _check(self._lib.tcrnet_edge_distances(self._ctx, C.byref(d)), "tcrnet_edge_distances")
        if not d.value:
            return torch.empty(0, dtype=torch.uint8, device=self.device)
        return self._view(d.value, torch.uint8, self.n_edges)

    def restrict(self, l_max: int) -> int:
        e = C.c_int64(0)
        _check(self._lib.tcrnet_restrict(self._ctx, int(l_max), C.byref(e)), "tcrnet_restrict")
        self.n_edges = int(e.value)
        return self.n_edges

    # -- network observables on the current CSR -------------------------
    def degree_histogram(self) -> "torch.Tensor":
        """tcrnet_degree_histogram: int64[max_degree + 1] (a view of library memory)."""
        h, m = C.c_void_p(), C.c_int32(0)
        _check(self._lib.tcrnet_degree_histogram(self._ctx, C.byref(h), C.byref(m)), "tcrnet_degree_histogram")
        return self._view(h.value, self._torch.int64, int(m.value) + 1)

    def neighbor_degree(self):
        """tcrnet_neighbor_degree: (nn_sum int64[n], class_sum int64[H], knn float64[H]) views, H = max degree + 1."""
        torch = self._torch
        hist_len = int(self.degree_histogram().numel())
        a, b, c = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(self._lib.tcrnet_neighbor_degree(self._ctx, C.byref(a), C.byref(b), C.byref(c)), "tcrnet_neighbor_degree")
        return (self._view(a.value, torch.int64, self.n), self._view(b.value, torch.int64, hist_len),
                self._view(c.value, torch.float64, hist_len))

    def components(self):
        """tcrnet_components: (label int32[n], comp_size int32[n], n_components, lcc)."""
        torch = self._torch
        a, b, nc, lcc = C.c_void_p(), C.c_void_p(), C.c_int64(0), C.c_int64(0)
        _check(self._lib.tcrnet_components(self._ctx, C.byref(a), C.byref(b), C.byref(nc), C.byref(lcc)),
               "tcrnet_components")
        return (self._view(a.value, torch.int32, self.n), self._view(b.value, torch.int32, self.n), int(nc.value),
                int(lcc.value))

    def percolation(self, removal_rank, n_removed, deg_hist: bool = False):
        """tcrnet_percolation: (lcc int64[K], lcc_norm1 float64[K], lcc_norm2 float64[K], deg_hist int64[K, H] or
        None) as numpy arrays; removal_rank is a host permutation of 0..n-1, n_removed the steps."""
        rank = np.ascontiguousarray(removal_rank, dtype=np.int32)
        steps = np.ascontiguousarray(n_removed, dtype=np.int64)
        if rank.size != self.n:
            raise TcrNetError(ERR_ARG, "tcrnet_percolation (removal_rank must have n entries)")
        k = int(steps.size)
        lcc = np.zeros(k, dtype=np.int64)
        n1 = np.zeros(k, dtype=np.float64)
        n2 = np.zeros(k, dtype=np.float64)
        hist = np.zeros((k, int(self.degree_histogram().numel())), dtype=np.int64) if deg_hist else None
        f64p = C.POINTER(C.c_double)
        _check(self._lib.tcrnet_percolation(
            self._ctx, rank.ctypes.data_as(C.POINTER(C.c_int32)), steps.ctypes.data_as(C.POINTER(C.c_int64)), k,
            lcc.ctypes.data_as(C.POINTER(C.c_int64)), n1.ctypes.data_as(f64p), n2.ctypes.data_as(f64p),
            hist.ctypes.data_as(C.POINTER(C.c_int64)) if hist is not None else None), "tcrnet_percolation")
        return lcc, n1, n2, hist

    def _view(self, ptr: int, dtype, count: int):
        """Zero-copy torch view of library-owned device memory (it was allocated by torch)."""
        block = self._blocks[ptr]
        return block.view(dtype)[:count]

    def csr(self) -> Tuple["torch.Tensor", "torch.Tensor"]:
        """(row_ptr int64[n+1], col int32[E]) — views valid until the next build/load/destroy."""
        torch = self._torch
        rp, cl = C.c_void_p(), C.c_void_p()
        _check(self._lib.tcrnet_csr(self._ctx, C.byref(rp), C.byref(cl)), "tcrnet_csr")
        row_ptr = self._view(rp.value, torch.int64, self.n + 1)
        col = (self._view(cl.value, torch.int32, self.n_edges) if cl.value
               else torch.empty(0, dtype=torch.int32, device=self.device))
        return row_ptr, col

    def degrees(self) -> "torch.Tensor":
        dg = C.c_void_p()
        _check(self._lib.tcrnet_degrees(self._ctx, C.byref(dg)), "tcrnet_degrees")
        return self._view(dg.value, self._torch.int32, self.n)

    def _host(self, name: str, count: int, dtype, staged: bool):
        if not staged:
            return np.empty(count, dtype=dtype)
        nbytes = max(count, 1) * np.dtype(dtype).itemsize
        t = self._staging.get(name)
        if t is None or t.numel() < nbytes:
            t = self._torch.empty(nbytes + nbytes // 4, dtype=self._torch.uint8, pin_memory=True)
            self._staging[name] = t
        return t.numpy()[:count * np.dtype(dtype).itemsize].view(dtype)

    def copy_csr(self, row_ptr: bool = True, col: bool = True, deg: bool = True, staged: bool = False):
        """tcrnet_copy_csr into numpy arrays: (row_ptr, col, deg) (None where skipped).

        staged=False: fresh pageable arrays.  staged=True: views of page-locked staging buffers
        owned by this object and reused by the next staged call (the device-to-host copy then runs
        at full PCIe rate; the caller must be done with them before calling again)."""
        rp = self._host("row_ptr", self.n + 1, np.int64, staged) if row_ptr else None
        cl = self._host("col", self.n_edges, np.int32, staged) if col else None
        dg = self._host("deg", self.n, np.int32, staged) if deg else None
        _check(self._lib.tcrnet_copy_csr(
            self._ctx,
            rp.ctypes.data_as(C.POINTER(C.c_int64)) if rp is not None else None,
            cl.ctypes.data_as(C.POINTER(C.c_int32)) if cl is not None and cl.size else None,
            dg.ctypes.data_as(C.POINTER(C.c_int32)) if dg is not None else None), "tcrnet_copy_csr")
        return rp, cl, dg

    def set_option(self, option: int, value: int) -> None:
        _check(self._lib.tcrnet_set_option(self._ctx, int(option), int(value)), "tcrnet_set_option")

    def get_stats(self) -> dict:
        st = tcrnet_stats()
        _check(self._lib.tcrnet_get_stats(self._ctx, C.byref(st)), "tcrnet_get_stats")
        return {name: getattr(st, name) for name, _ in tcrnet_stats._fields_}

    def probe_int32(self, kind: int) -> Tuple[float, float]:
        ops, mhz = C.c_double(0), C.c_double(0)
        _check(self._lib.tcrnet_probe_int32(self._ctx, int(kind), C.byref(ops), C.byref(mhz)), "tcrnet_probe_int32")
        return float(ops.value), float(mhz.value)

    def last_cuda_error(self) -> int:
        return int(self._lib.tcrnet_last_cuda_error(self._ctx))


def row_ptr_noalloc(counts, row_ptr, n: Optional[int] = None, stream=None) -> None:
    """tcrnet_row_ptr_noalloc: row_ptr[0] = 0, row_ptr[u + 1] = row_ptr[u] + counts[u], enqueued on `stream` (default:
    torch's current stream of the tensors' device) - no allocation here or in the library, no synchronisation.
    counts: int32 CUDA tensor (>= n elements), row_ptr: int64 CUDA tensor (>= n + 1 elements), both the caller's."""
    import torch
    assert counts.is_cuda and row_ptr.is_cuda and counts.device == row_ptr.device
    assert counts.dtype == torch.int32 and row_ptr.dtype == torch.int64
    assert counts.is_contiguous() and row_ptr.is_contiguous()
    n = int(counts.numel()) if n is None else int(n)
    if 0 <= n <= NOALLOC_MAX_ROWS:  # (beyond the capacity the library refuses before it looks at a pointer)
        assert counts.numel() >= n and row_ptr.numel() >= n + 1
    lib = load_library()
    err = C.c_int(0)
    with torch.cuda.device(counts.device):
        s = stream if stream is not None else torch.cuda.current_stream(counts.device)
        status = lib.tcrnet_row_ptr_noalloc(C.c_void_p(counts.data_ptr()), n, C.c_void_p(row_ptr.data_ptr()),
                                            C.c_void_p(s.cuda_stream), C.byref(err))
    if status != OK:
        raise TcrNetError(status, "tcrnet_row_ptr_noalloc" + (f" (cudaError {err.value})" if err.value else ""))


def build_network(residues, lengths, l_max: int, device: int = 0):
    """Convenience: load + build + copy back.  Returns (row_ptr, col, deg) as numpy arrays."""
    with TcrNet(device) as net:
        net.load(residues, lengths)
        net.build(l_max)
        return net.copy_csr()
