"""CPU oracle for the TCR-NET hot path — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA
package and shares no code with it.  The arithmetic lives in
``oracle/tcrnet_oracle.c`` (plain Wagner-Fischer + double loop + counting; every
function cites the passage of PAPER.md it follows); this module only marshals
numpy arrays into it through ctypes.  The network observables of SURVEY 8(f) NEXT-1 (degree
distribution, average neighbour degree, connected components / LCC, site percolation) live in
``oracle/network_oracle.c`` and are pinned by tests/test_observables_pins.py.

Parity status: every function is pinned (tests/test_oracle_pins.py); nothing here
is "parity unpinned".
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence, Tuple

import numpy as np

from .build import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build())
        u8p, i32p, i64p = C.POINTER(C.c_uint8), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        lib.oracle_lev.restype = C.c_int32
        lib.oracle_lev.argtypes = [u8p, C.c_int32, u8p, C.c_int32]
        lib.oracle_lev_abort.restype = C.c_int32
        lib.oracle_lev_abort.argtypes = [u8p, C.c_int32, u8p, C.c_int32, C.c_int32]
        lib.oracle_edges.restype = C.c_int
        lib.oracle_edges.argtypes = [u8p, i64p, i32p, C.c_int64, C.c_int32, i64p, C.c_int64, C.c_int,
                                     C.c_int, C.c_int, C.POINTER(i64p), i64p, i32p]
        lib.oracle_lev_pairs.restype = C.c_int
        lib.oracle_lev_pairs.argtypes = [u8p, i64p, i32p, C.c_int64, i64p, C.c_int64, i32p, C.c_int]
        lib.oracle_free.restype = None
        lib.oracle_free.argtypes = [C.c_void_p]
        lib.oracle_csr.restype = C.c_int
        lib.oracle_csr.argtypes = [i64p, C.c_int64, C.c_int64, i64p, i32p, i32p]
        f64p = C.POINTER(C.c_double)
        lib.oracle_degree_histogram.restype = C.c_int64
        lib.oracle_degree_histogram.argtypes = [i32p, C.c_int64, i64p, C.c_int64]
        lib.oracle_neighbor_degree.restype = C.c_int
        lib.oracle_neighbor_degree.argtypes = [i64p, i32p, C.c_int64, i64p, i64p, f64p, C.c_int64]
        lib.oracle_components.restype = C.c_int
        lib.oracle_components.argtypes = [i64p, i32p, C.c_int64, u8p, i32p, i32p, i64p, i64p]
        lib.oracle_percolation.restype = C.c_int
        lib.oracle_percolation.argtypes = [i64p, i32p, C.c_int64, i32p, i64p, C.c_int64, i64p, f64p, f64p, i64p,
                                           C.c_int64]
        _lib = lib
    return _lib


def _u8(x) -> np.ndarray:
    if isinstance(x, str):
        x = x.encode()
    if isinstance(x, (bytes, bytearray)):
        return np.frombuffer(bytes(x), dtype=np.uint8)
    return np.ascontiguousarray(x, dtype=np.uint8)


def _ptr(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def lev(a, b) -> int:
    """Unit-cost Levenshtein distance, full Wagner-Fischer table."""
    a, b = _u8(a), _u8(b)
    d = _load().oracle_lev(_ptr(a, C.c_uint8), a.size, _ptr(b, C.c_uint8), b.size)
    if d < 0:
        raise MemoryError("oracle_lev")
    return int(d)


def lev_abort(a, b, l_max: int) -> int:
    """Same, with the paper's row-minimum abort; returns l_max+1 when aborted."""
    a, b = _u8(a), _u8(b)
    d = _load().oracle_lev_abort(_ptr(a, C.c_uint8), a.size, _ptr(b, C.c_uint8), b.size, int(l_max))
    if d < 0:
        raise MemoryError("oracle_lev_abort")
    return int(d)


def _offsets(lengths: np.ndarray) -> np.ndarray:
    off = np.zeros(lengths.size + 1, dtype=np.int64)
    np.cumsum(lengths, out=off[1:])
    return off


def edges(residues, lengths, l_max: int, *, rows: Optional[Sequence[int]] = None,
          all_partners: bool = False, tier: int = 0, threads: int = 0) -> Tuple[np.ndarray, int]:
    """Pairs (i, j) with lev(s_i, s_j) <= l_max, loop order.

    Returns (int64[E, 2], threads_used).  ``rows`` restricts the first index;
    ``all_partners`` makes j range over every row != i instead of j > i.
    """
    residues = _u8(residues)
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    off = _offsets(lengths)
    assert off[-1] == residues.size, "residues / lengths mismatch"
    rows_arr = None
    if rows is not None:
        rows_arr = np.ascontiguousarray(rows, dtype=np.int64)
    out = C.POINTER(C.c_int64)()
    n_out = C.c_int64(0)
    used = C.c_int32(0)
    rc = _load().oracle_edges(
        _ptr(residues, C.c_uint8), _ptr(off, C.c_int64), _ptr(lengths, C.c_int32), lengths.size, int(l_max),
        _ptr(rows_arr, C.c_int64) if rows_arr is not None else None,
        rows_arr.size if rows_arr is not None else 0, int(all_partners), int(tier), int(threads),
        C.byref(out), C.byref(n_out), C.byref(used))
    if rc != 0:
        raise MemoryError("oracle_edges")
    e = n_out.value
    pairs = np.ctypeslib.as_array(out, shape=(max(e, 1) * 2,))[: 2 * e].copy().reshape(e, 2)
    _load().oracle_free(out)
    return pairs, int(used.value)


def lev_pairs(residues, lengths, pairs, *, threads: int = 0) -> np.ndarray:
    """lev(s_i, s_j) (full table) for every (i, j) of ``pairs`` (int64[E, 2]): int32[E]."""
    residues = _u8(residues)
    lengths = np.ascontiguousarray(lengths, dtype=np.int32)
    off = _offsets(lengths)
    assert off[-1] == residues.size, "residues / lengths mismatch"
    pairs = np.ascontiguousarray(pairs, dtype=np.int64).reshape(-1, 2)
    out = np.zeros(pairs.shape[0], dtype=np.int32)
    rc = _load().oracle_lev_pairs(_ptr(residues, C.c_uint8), _ptr(off, C.c_int64), _ptr(lengths, C.c_int32),
                                  lengths.size, _ptr(pairs, C.c_int64), pairs.shape[0], _ptr(out, C.c_int32),
                                  int(threads))
    if rc != 0:
        raise ValueError("oracle_lev_pairs: index out of range or out of memory")
    return out


def csr(pairs: np.ndarray, n: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """(row_ptr int64[n+1], col int32[E], deg int32[n]) from sorted (i<j) pairs.

    PAPER.md:301-318 (adjacency, upper triangle) and PAPER.md:224 (degree).
    """
    pairs = np.ascontiguousarray(pairs, dtype=np.int64).reshape(-1, 2)
    e = pairs.shape[0]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    col = np.zeros(e, dtype=np.int32)
    deg = np.zeros(n, dtype=np.int32)
    rc = _load().oracle_csr(_ptr(pairs, C.c_int64), e, n, _ptr(row_ptr, C.c_int64), _ptr(col, C.c_int32),
                            _ptr(deg, C.c_int32))
    if rc != 0:
        raise ValueError("oracle_csr: pairs must be strictly increasing (i<j) and in range")
    return row_ptr, col, deg


def network(residues, lengths, l_max: int, *, tier: int = 0, threads: int = 0):
    """The whole path: (row_ptr, col, deg, threads_used)."""
    pairs, used = edges(residues, lengths, l_max, tier=tier, threads=threads)
    n = int(np.asarray(lengths).size)
    row_ptr, col, deg = csr(pairs, n)
    return row_ptr, col, deg, used


# ---- network observables on the CSR (oracle/network_oracle.c) ------------------------------------

def _csr_args(row_ptr, col):
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col = np.ascontiguousarray(col, dtype=np.int32)
    n = row_ptr.size - 1
    assert n >= 0 and row_ptr[0] == 0 and int(row_ptr[-1]) == col.size
    if col.size == 0:
        col = np.zeros(1, dtype=np.int32)  # a valid pointer for ctypes; never read
    return row_ptr, col, n


def degree_histogram(deg) -> np.ndarray:
    """hist[d] = number of nodes of degree d, d = 0..max degree (p_d = hist[d] / N)."""
    deg = np.ascontiguousarray(deg, dtype=np.int32)
    hist_len = int(deg.max()) + 1 if deg.size else 1
    hist = np.zeros(hist_len, dtype=np.int64)
    rc = _load().oracle_degree_histogram(_ptr(deg, C.c_int32), deg.size, _ptr(hist, C.c_int64), hist_len)
    if rc < 0:
        raise ValueError("oracle_degree_histogram")
    return hist


def neighbor_degree(row_ptr, col, hist_len: int):
    """(nn_sum int64[n], class_sum int64[hist_len], knn float64[hist_len]): Eq. 9."""
    row_ptr, col, n = _csr_args(row_ptr, col)
    nn_sum = np.zeros(max(n, 1), dtype=np.int64)
    class_sum = np.zeros(hist_len, dtype=np.int64)
    knn = np.zeros(hist_len, dtype=np.float64)
    rc = _load().oracle_neighbor_degree(_ptr(row_ptr, C.c_int64), _ptr(col, C.c_int32), n, _ptr(nn_sum, C.c_int64),
                                        _ptr(class_sum, C.c_int64), _ptr(knn, C.c_double), hist_len)
    if rc != 0:
        raise ValueError(f"oracle_neighbor_degree rc={rc}")
    return nn_sum[:n], class_sum, knn


def components(row_ptr, col, alive=None):
    """(label int32[n], comp_size int32[n], n_components, lcc): PAPER.md:224; label = smallest node id of the
    component, -1 / size 0 for removed nodes (alive[u] == 0)."""
    row_ptr, col, n = _csr_args(row_ptr, col)
    label = np.zeros(max(n, 1), dtype=np.int32)
    size = np.zeros(max(n, 1), dtype=np.int32)
    al = None
    if alive is not None:
        al = np.ascontiguousarray(alive, dtype=np.uint8)
        assert al.size == n
    nc, lcc = C.c_int64(0), C.c_int64(0)
    rc = _load().oracle_components(_ptr(row_ptr, C.c_int64), _ptr(col, C.c_int32), n,
                                   _ptr(al, C.c_uint8) if al is not None else None, _ptr(label, C.c_int32),
                                   _ptr(size, C.c_int32), C.byref(nc), C.byref(lcc))
    if rc != 0:
        raise MemoryError("oracle_components")
    return label[:n], size[:n], int(nc.value), int(lcc.value)


def percolation(row_ptr, col, removal_rank, n_removed, hist_len: int = 0):
    """Site percolation along one removal order:
    (lcc int64[K], lcc_norm1 float64[K] (Eq. 12), lcc_norm2 float64[K] (Eq. 13), deg_hist int64[K, hist_len] or None)."""
    row_ptr, col, n = _csr_args(row_ptr, col)
    rank = np.ascontiguousarray(removal_rank, dtype=np.int32)
    steps = np.ascontiguousarray(n_removed, dtype=np.int64)
    assert rank.size == n
    k = steps.size
    lcc = np.zeros(max(k, 1), dtype=np.int64)
    n1 = np.zeros(max(k, 1), dtype=np.float64)
    n2 = np.zeros(max(k, 1), dtype=np.float64)
    hist = np.zeros((max(k, 1), hist_len), dtype=np.int64) if hist_len > 0 else None
    rc = _load().oracle_percolation(_ptr(row_ptr, C.c_int64), _ptr(col, C.c_int32), n, _ptr(rank, C.c_int32),
                                    _ptr(steps, C.c_int64), k, _ptr(lcc, C.c_int64), _ptr(n1, C.c_double),
                                    _ptr(n2, C.c_double), _ptr(hist, C.c_int64) if hist is not None else None,
                                    hist_len)
    if rc != 0:
        raise ValueError(f"oracle_percolation rc={rc}")
    return lcc[:k], n1[:k], n2[:k], (hist[:k] if hist is not None else None)
