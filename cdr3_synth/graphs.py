"""Seeded random graphs with the shape of a TCR network, as plain edge lists.

Inputs for the parity tests of the network observables at sizes where the
oracle cannot build the Levenshtein network itself (N = 800,000 takes core-hours): the CUDA path
takes the edge list through ``tcrnet_assemble``, the oracle through ``oracle.csr``.  Like the
rest of this package the module holds none of the method's arithmetic (no degrees, no components,
no percolation) - only random draws, sorting and de-duplication of index pairs.

Recipe (``family_graph``), every draw from ``numpy.random.Generator(PCG64(seed))`` in this order:
1. family sizes ``Poisson(lam) + 1`` until they cover ``round((1 - isolated) * n)`` nodes (last one
   cut); the remaining nodes have no family;
2. inside a family of size s: ``ceil(density * s * (s - 1) / 2)`` node pairs drawn uniformly with
   replacement (duplicates and loops dropped) - dense clusters, as the variants of one seed are;
3. ``round(bridges * n)`` pairs of uniformly drawn family nodes - the sparse links that join
   clusters into a large component;
4. one uniform random relabelling of the n nodes (families are not index-contiguous);
5. pairs are oriented i < j, de-duplicated and sorted lexicographically.
Measured shape at the defaults (n = 800,000, seed 1): 3.44 M edges, mean degree 8.6, maximum degree 25,
32,693 components, a largest component of 61 % of the nodes, 3 % isolated nodes - the scale of
config 4's network (4.36 M edges).
"""
from __future__ import annotations

import numpy as np


def family_graph(n: int, seed: int, lam: float = 24.0, density: float = 0.45, bridges: float = 0.03,
                 isolated: float = 0.03) -> np.ndarray:
    """int64[E, 2] sorted (i < j) edge list on nodes 0..n-1."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n_fam_nodes = int(round((1.0 - isolated) * n))
    sizes = []
    total = 0
    while total < n_fam_nodes:
        chunk = rng.poisson(lam, size=max(16, n_fam_nodes // int(lam + 1) + 16)) + 1
        for s in chunk.tolist():
            if total >= n_fam_nodes:
                break
            s = min(s, n_fam_nodes - total)
            sizes.append(s)
            total += s
    sizes = np.asarray(sizes, dtype=np.int64)
    starts = np.concatenate([[0], np.cumsum(sizes)[:-1]])
    m = np.ceil(density * sizes * (sizes - 1) / 2.0).astype(np.int64)
    fam = np.repeat(np.arange(sizes.size), m)
    a = starts[fam] + (rng.random(fam.size) * sizes[fam]).astype(np.int64)
    b = starts[fam] + (rng.random(fam.size) * sizes[fam]).astype(np.int64)
    nb = int(round(bridges * n))
    a = np.concatenate([a, rng.integers(0, max(n_fam_nodes, 1), size=nb)])
    b = np.concatenate([b, rng.integers(0, max(n_fam_nodes, 1), size=nb)])
    relabel = rng.permutation(n).astype(np.int64)
    a, b = relabel[a], relabel[b]
    lo, hi = np.minimum(a, b), np.maximum(a, b)
    keep = lo != hi
    keys = np.unique(lo[keep] * np.int64(n) + hi[keep])
    return np.stack([keys // n, keys % n], axis=1).astype(np.int64)
