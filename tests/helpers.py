"""Shared helpers of the parity tests (comparison logic only; no method arithmetic)."""
from __future__ import annotations

import numpy as np


def csr_rows(row_ptr: np.ndarray) -> np.ndarray:
    """First index of every edge of a CSR (expanded row ids)."""
    return np.repeat(np.arange(row_ptr.size - 1, dtype=np.int64), np.diff(row_ptr))


def check_csr_invariants(row_ptr, col, deg, n):
    """Properties that hold at any size: shapes, monotone row_ptr, strict upper triangle, strictly
    ascending columns per row, sum(deg) = 2E, deg = upper count + lower count."""
    assert row_ptr.shape == (n + 1,) and deg.shape == (n,)
    e = int(row_ptr[-1])
    assert row_ptr[0] == 0 and col.shape == (e,)
    assert (np.diff(row_ptr) >= 0).all()
    rows = csr_rows(row_ptr)
    assert (col > rows).all() and (col < n).all()
    same_row = rows[1:] == rows[:-1]
    assert (np.diff(col.astype(np.int64))[same_row] > 0).all()
    assert int(deg.astype(np.int64).sum()) == 2 * e
    want = np.bincount(rows, minlength=n) + np.bincount(col, minlength=n)
    assert np.array_equal(want, deg)


def neighbours_from_csr(row_ptr, col, nodes):
    """Full neighbourhood (both directions) of each node in `nodes`, ascending."""
    rows = csr_rows(row_ptr)
    out = {}
    for u in nodes:
        upper = col[row_ptr[u]:row_ptr[u + 1]].astype(np.int64)
        lower = rows[col == u]
        out[int(u)] = np.sort(np.concatenate([lower, upper]))
    return out


def neighbours_from_pairs(pairs, nodes):
    """Same from the oracle's (i, j) list produced with all_partners=True."""
    return {int(u): np.sort(pairs[pairs[:, 0] == u, 1]) for u in nodes}


def assert_same_network(got, want):
    (rp, cl, dg), (orp, ocl, odg) = got, want
    assert int(rp[-1]) == int(orp[-1]), f"edge count {int(rp[-1])} != oracle {int(orp[-1])}"
    assert np.array_equal(rp, orp), "row_ptr differs"
    assert np.array_equal(cl, ocl), "col differs"
    assert np.array_equal(dg, odg), "deg differs"
