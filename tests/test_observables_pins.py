"""Pins of the observables oracle (oracle/network_oracle.c) against things other than
itself: networkx (the library the paper used) and scipy.sparse.csgraph as independent library
routines, closed forms, the paper's 5-node example, brute-force reachability on tiny graphs.
CPU only."""
from __future__ import annotations

import os

import networkx as nx
import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components

import oracle


def csr_from_edges(n, edges):
    """Strict-upper-triangle CSR of an undirected simple graph given as (u, v) pairs (test helper: sorting and
    counting only)."""
    e = sorted({(min(u, v), max(u, v)) for u, v in edges if u != v})
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    for u, _ in e:
        row_ptr[u + 1] += 1
    row_ptr = np.cumsum(row_ptr)
    col = np.array([v for _, v in e], dtype=np.int32)
    return row_ptr, col, e


def random_graph(rng, n, m):
    edges = set()
    while len(edges) < m:
        u, v = int(rng.integers(n)), int(rng.integers(n))
        if u != v:
            edges.add((min(u, v), max(u, v)))
    return sorted(edges)


def nx_graph(n, e):
    g = nx.Graph()
    g.add_nodes_from(range(n))
    g.add_edges_from(e)
    return g


def degrees(n, e):
    d = np.zeros(n, dtype=np.int32)
    for u, v in e:
        d[u] += 1
        d[v] += 1
    return d


def test_paper_five_node_example(golden_dir):
    vals = {}
    for line in open(os.path.join(golden_dir, "paper_adjacency_example.txt")):
        if line.startswith("#") or ":" not in line:
            continue
        k, v = line.split(":")
        vals[k.strip()] = [int(x) for x in v.split()]
    e1 = vals["edges_1based"]
    edges = [(e1[i] - 1, e1[i + 1] - 1) for i in range(0, len(e1), 2)]
    row_ptr, col, _ = csr_from_edges(5, edges)
    assert list(row_ptr) == vals["row_ptr"] and list(col) == vals["col"]
    deg = np.array(vals["deg"], dtype=np.int32)
    assert list(oracle.degree_histogram(deg)) == vals["deg_hist"]
    nn_sum, class_sum, knn = oracle.neighbor_degree(row_ptr, col, 3)
    assert list(nn_sum) == vals["nn_sum"] and list(class_sum) == vals["class_sum"]
    nd = vals["knn_num_den"]
    assert knn[0] == 0.0 and knn[1] == nd[2] / nd[3] and knn[2] == nd[4] / nd[5]
    label, size, ncomp, lcc = oracle.components(row_ptr, col)
    assert ncomp == vals["components"][0] and lcc == vals["lcc"][0]
    assert list(label) == [0] * 5 and list(size) == [5] * 5


@pytest.mark.parametrize("n,m,seed", [(1, 0, 0), (2, 0, 1), (2, 1, 2), (40, 25, 3), (200, 150, 4), (300, 900, 5),
                                      (1000, 700, 6)])
def test_against_networkx_and_scipy(n, m, seed):
    rng = np.random.default_rng(seed)
    e = random_graph(rng, n, m)
    row_ptr, col, _ = csr_from_edges(n, e)
    g = nx_graph(n, e)
    deg = degrees(n, e)
    # degree distribution
    assert list(oracle.degree_histogram(deg)) == nx.degree_histogram(g)
    # neighbour degrees (Eq. 9): per node and per degree class
    hist_len = int(deg.max()) + 1
    nn_sum, class_sum, knn = oracle.neighbor_degree(row_ptr, col, hist_len)
    per_node = nx.average_neighbor_degree(g)
    for u in range(n):
        want = per_node[u]
        got = nn_sum[u] / deg[u] if deg[u] else 0.0
        assert got == pytest.approx(want, rel=1e-12, abs=0)
    per_class = nx.average_degree_connectivity(g)
    for d in range(hist_len):
        if d in per_class:
            assert knn[d] == pytest.approx(per_class[d], rel=1e-12, abs=0)
        else:
            assert knn[d] == 0.0
    # components: networkx sets, scipy labels
    label, size, ncomp, lcc = oracle.components(row_ptr, col)
    comps = list(nx.connected_components(g))
    assert ncomp == len(comps) and lcc == max(len(c) for c in comps)
    for c in comps:
        for u in c:
            assert label[u] == min(c) and size[u] == len(c)
    a = sp.coo_matrix((np.ones(len(e)), ([u for u, _ in e], [v for _, v in e])), shape=(n, n))
    k, lab = connected_components(a, directed=False)
    assert k == ncomp
    # same partition: scipy's labels are constant exactly where ours are
    assert len(set(zip(lab.tolist(), label.tolist()))) == k


def _reach_closure(n, e):
    r = np.eye(n, dtype=bool)
    for u, v in e:
        r[u, v] = r[v, u] = True
    for _ in range(n):  # boolean matrix "squaring" until fixed point: brute-force reachability
        r2 = (r.astype(np.int32) @ r.astype(np.int32)) > 0
        if (r2 == r).all():
            break
        r = r2
    return r


@pytest.mark.parametrize("seed", range(6))
def test_components_brute_force_reachability(seed):
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(2, 14))
    e = random_graph(rng, n, int(rng.integers(0, min(12, n * (n - 1) // 2) + 1)))
    alive = rng.random(n) < 0.75
    row_ptr, col, _ = csr_from_edges(n, e)
    label, size, ncomp, lcc = oracle.components(row_ptr, col, alive)
    e_alive = [(u, v) for u, v in e if alive[u] and alive[v]]
    r = _reach_closure(n, e_alive)
    seen = set()
    for u in range(n):
        if not alive[u]:
            assert label[u] == -1 and size[u] == 0
            continue
        members = [v for v in range(n) if alive[v] and r[u, v]]
        assert label[u] == min(members) and size[u] == len(members)
        seen.add(min(members))
    assert ncomp == len(seen)
    assert lcc == (max(size) if alive.any() else 0)


def test_closed_forms():
    # path P_n: one component; <d_nn>(1) = 2, <d_nn>(2) = (2*3 + (n-4)*4) / (2 (n-2)) for n >= 4
    n = 50
    rp, col, e = csr_from_edges(n, [(i, i + 1) for i in range(n - 1)])
    _, _, ncomp, lcc = oracle.components(rp, col)
    assert (ncomp, lcc) == (1, n)
    _, class_sum, knn = oracle.neighbor_degree(rp, col, 3)
    assert knn[1] == 2.0 and knn[2] == (2 * 3 + (n - 4) * 4) / (2 * (n - 2))
    # star K_{1,r}: leaves see the centre (degree r), the centre sees leaves (degree 1)
    r = 17
    rp, col, e = csr_from_edges(r + 1, [(0, i) for i in range(1, r + 1)])
    nn_sum, class_sum, knn = oracle.neighbor_degree(rp, col, r + 1)
    assert knn[1] == float(r) and knn[r] == 1.0 and nn_sum[0] == r and all(nn_sum[1:] == r)
    assert list(oracle.degree_histogram(degrees(r + 1, e))) == [0, r] + [0] * (r - 2) + [1]
    # complete graph K_r plus isolated nodes: r-clique is the LCC, isolated nodes are components of size 1
    k, iso = 9, 4
    rp, col, e = csr_from_edges(k + iso, [(i, j) for i in range(k) for j in range(i + 1, k)])
    label, size, ncomp, lcc = oracle.components(rp, col)
    assert (ncomp, lcc) == (1 + iso, k) and list(label[k:]) == list(range(k, k + iso))
    _, _, knn = oracle.neighbor_degree(rp, col, k)
    assert knn[k - 1] == float(k - 1) and knn[0] == 0.0  # reading Q15
    # two disjoint cycles C_a, C_b
    a, b = 5, 8
    ed = [(i, (i + 1) % a) for i in range(a)] + [(a + i, a + (i + 1) % b) for i in range(b)]
    rp, col, e = csr_from_edges(a + b, ed)
    label, size, ncomp, lcc = oracle.components(rp, col)
    assert (ncomp, lcc) == (2, b) and set(label[:a]) == {0} and set(label[a:]) == {a}
    # empty graph
    rp, col, e = csr_from_edges(6, [])
    label, size, ncomp, lcc = oracle.components(rp, col)
    assert (ncomp, lcc) == (6, 1) and list(label) == list(range(6))


def test_percolation_closed_forms_and_networkx():
    # path 0-1-2-...-9, remove from the left end: LCC = what is left; remove the middle node first: halves
    n = 10
    rp, col, e = csr_from_edges(n, [(i, i + 1) for i in range(n - 1)])
    rank = np.arange(n, dtype=np.int32)
    lcc, n1, n2, hist = oracle.percolation(rp, col, rank, np.arange(n + 1), hist_len=3)
    assert list(lcc) == list(range(n, -1, -1))
    assert list(n1[:-1]) == [1.0] * n and n1[-1] == 0.0 and list(n2[:-1]) == [1.0] * n  # Eq. 12, 13; Q16
    assert list(hist[0]) == [0, 2, n - 2] and list(hist[n - 1]) == [1, 0, 0] and list(hist[n]) == [0, 0, 0]
    rank = np.array([1, 2, 3, 4, 0, 5, 6, 7, 8, 9], dtype=np.int32)  # node 4 goes first
    lcc, n1, n2, _ = oracle.percolation(rp, col, rank, [0, 1])
    assert list(lcc) == [10, 5] and n1[1] == 5 / 9 and n2[1] == (5 / 9) / 1.0
    # star: removing the centre first shatters it
    r = 12
    rp, col, e = csr_from_edges(r + 1, [(0, i) for i in range(1, r + 1)])
    lcc, _, _, _ = oracle.percolation(rp, col, np.arange(r + 1, dtype=np.int32), [0, 1, 2])
    assert list(lcc) == [r + 1, 1, 1]
    # random graph, random order: every step against networkx on the induced subgraph
    rng = np.random.default_rng(7)
    n = 400
    e = random_graph(rng, n, 500)
    rp, col, _ = csr_from_edges(n, e)
    g = nx_graph(n, e)
    rank = rng.permutation(n).astype(np.int32)
    steps = [0, 1, 13, 100, 250, 399, 400, 57]  # any order of steps
    deg = degrees(n, e)
    lcc, n1, n2, hist = oracle.percolation(rp, col, rank, steps, hist_len=int(deg.max()) + 1)
    lcc0 = max(len(c) for c in nx.connected_components(g))
    for k, nr in enumerate(steps):
        sub = g.subgraph([u for u in range(n) if rank[u] >= nr])
        want = max((len(c) for c in nx.connected_components(sub)), default=0)
        assert lcc[k] == want
        assert n1[k] == (want / (n - nr) if n > nr else 0.0)
        assert n2[k] == (n1[k] / (lcc0 / n))
        h = nx.degree_histogram(sub)
        assert list(hist[k][:len(h)]) == h and not hist[k][len(h):].any()
    # not a permutation -> error
    with pytest.raises(ValueError):
        oracle.percolation(rp, col, np.zeros(n, dtype=np.int32), [0])


def test_observables_on_a_tcr_network():
    """The oracle's own cfg1 network (l_max = 1) against networkx end to end."""
    from cdr3_synth import generate
    d = generate("cfg1")
    row_ptr, col, deg, _ = oracle.network(d.residues, d.lengths, 1, tier=1)
    rows = np.repeat(np.arange(d.n), np.diff(row_ptr))
    g = nx_graph(d.n, list(zip(rows.tolist(), col.tolist())))
    assert list(oracle.degree_histogram(deg)) == nx.degree_histogram(g)
    label, size, ncomp, lcc = oracle.components(row_ptr, col)
    comps = list(nx.connected_components(g))
    assert ncomp == len(comps) and lcc == max(map(len, comps))
    _, _, knn = oracle.neighbor_degree(row_ptr, col, int(deg.max()) + 1)
    for dd, v in nx.average_degree_connectivity(g).items():
        assert knn[dd] == pytest.approx(v, rel=1e-12, abs=0)
