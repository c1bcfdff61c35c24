"""Parity of the network observables computed by the CUDA path, through the C ABI,
against the CPU oracle (oracle/network_oracle.c): element by element, bit-exact - integers, and doubles
that are one IEEE division of two integers on both sides.

cfg1 / cfg2: the oracle builds the Levenshtein network itself and the CUDA path builds its own; at
N = 800,000 (the size the paper analyses, Fig. 2(f)-(h)) both sides take the same seeded synthetic
edge list (cdr3_synth.graphs), the CUDA path through tcrnet_assemble.  No oracle input comes from the
CUDA path.
"""
import numpy as np
import pytest

from cdr3_synth import generate
from cdr3_synth.generator import from_strings
from cdr3_synth.graphs import family_graph

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2112_06613_b200 as p
    return p


@pytest.fixture(scope="module")
def oracle():
    import oracle as o
    return o


def steps_for(n, k=11):
    s = np.unique(np.concatenate([(np.linspace(0.0, 1.0, k) * n).astype(np.int64), [0, 1, n - 1, n]]))
    return s[(s >= 0) & (s <= n)][::-1].copy()  # descending: any order of steps is allowed


def check_all_observables(net, oracle, row_ptr, col, deg, seed, n_steps=11):
    """net holds a built network whose CSR the caller has already checked to equal (row_ptr, col, deg)."""
    n = deg.size
    # degree distribution
    hist = net.degree_histogram().cpu().numpy()
    want_hist = oracle.degree_histogram(deg)
    assert np.array_equal(hist, want_hist)
    assert hist.sum() == n and (np.arange(hist.size) * hist).sum() == 2 * col.size
    # neighbour degrees, Eq. 9
    nn, cs, knn = (t.cpu().numpy() for t in net.neighbor_degree())
    o_nn, o_cs, o_knn = oracle.neighbor_degree(row_ptr, col, hist.size)
    assert np.array_equal(nn, o_nn) and np.array_equal(cs, o_cs)
    assert np.array_equal(knn, o_knn), "knn differs (must be bit-equal: one IEEE division)"
    # components
    label, size, ncomp, lcc = net.components()
    o_label, o_size, o_ncomp, o_lcc = oracle.components(row_ptr, col)
    assert (ncomp, lcc) == (o_ncomp, o_lcc)
    assert np.array_equal(label.cpu().numpy(), o_label) and np.array_equal(size.cpu().numpy(), o_size)
    # percolation along one seeded removal order
    rank = np.random.default_rng(seed).permutation(n).astype(np.int32)
    steps = steps_for(n, n_steps)
    got = net.percolation(rank, steps, deg_hist=True)
    want = oracle.percolation(row_ptr, col, rank, steps, hist_len=hist.size)
    for g, w, name in zip(got, want, ("lcc", "norm1", "norm2", "deg_hist")):
        assert np.array_equal(g, w), name
    # without the histograms, same LCCs
    got2 = net.percolation(rank, steps)
    assert got2[3] is None and np.array_equal(got2[0], want[0])
    return want


@pytest.mark.parametrize("name,l_max", [("cfg1", 1), ("cfg1", 3), ("cfg2", 1), ("cfg2", 2)])
def test_observables_of_the_levenshtein_network(pkg, oracle, name, l_max):
    d = generate(name)
    row_ptr, col, deg, _ = oracle.network(d.residues, d.lengths, l_max, tier=1)
    with pkg.TcrNet(0) as net:
        net.load(d.residues, d.lengths)
        net.build(l_max)
        rp, cl, dg = net.copy_csr()
        assert np.array_equal(rp, row_ptr) and np.array_equal(cl, col) and np.array_equal(dg, deg)
        check_all_observables(net, oracle, row_ptr, col, deg, seed=11)


def test_observables_at_paper_scale_on_a_synthetic_graph(pkg, oracle):
    """N = 800,000 nodes, 3.4 M edges (the scale of Fig. 2(f)-(h)); edge list -> tcrnet_assemble."""
    import torch
    n = 800_000
    pairs = family_graph(n, seed=1)
    row_ptr, col, deg = oracle.csr(pairs, n)
    d = generate("cfg4")  # any n loaded rows: assemble only needs the node count
    keys = torch.from_numpy((pairs[:, 0] << 32) | pairs[:, 1])
    keys = keys[torch.from_numpy(np.random.default_rng(3).permutation(keys.numel()))].cuda()  # any order
    with pkg.TcrNet(0) as net:
        net.load(d.residues, d.lengths)
        assert net.assemble(keys) == pairs.shape[0]
        rp, cl, dg = net.copy_csr()
        assert np.array_equal(rp, row_ptr) and np.array_equal(cl, col) and np.array_equal(dg, deg)
        lcc, n1, n2, _ = check_all_observables(net, oracle, row_ptr, col, deg, seed=12, n_steps=21)
    assert lcc[-1] > n // 2 and (np.diff(lcc) >= 0).all()  # steps descend in n_removed: nested removal


def test_headline_network_properties(pkg):
    """cfg4 (N = 800,000, l_max = 1), the network bench.py builds: properties that hold at any size."""
    d = generate("cfg4")
    with pkg.TcrNet(0) as net:
        net.load(d.residues, d.lengths)
        e = net.build(1)
        rp, cl, dg = net.copy_csr()
        hist = net.degree_histogram().cpu().numpy()
        assert np.array_equal(hist, np.bincount(dg, minlength=hist.size))
        nn, cs, knn = (t.cpu().numpy() for t in net.neighbor_degree())
        assert nn.sum() == (dg.astype(np.int64) ** 2).sum()  # every node contributes d(u) to each neighbour
        assert np.array_equal(cs, np.bincount(dg, weights=nn, minlength=hist.size).astype(np.int64))
        label, size, ncomp, lcc = net.components()
        label, size = label.cpu().numpy(), size.cpu().numpy()
        roots = np.nonzero(label == np.arange(d.n))[0]
        assert roots.size == ncomp and size[roots].sum() == d.n and size.max() == lcc
        assert (label <= np.arange(d.n)).all() and np.array_equal(label[label], label)
        rows = np.repeat(np.arange(d.n), np.diff(rp))
        assert np.array_equal(label[rows], label[cl])  # both ends of an edge share a label
        assert np.array_equal(size, np.bincount(label, minlength=d.n)[label])
        rank = np.random.default_rng(5).permutation(d.n).astype(np.int32)
        steps = (np.linspace(0, 1, 51) * d.n).astype(np.int64)
        p_lcc, n1, n2, h = net.percolation(rank, steps, deg_hist=True)
        assert p_lcc[0] == lcc and n2[0] == 1.0 and p_lcc[-1] == 0 and (np.diff(p_lcc) <= 0).all()
        assert np.array_equal(h[0], hist) and np.array_equal(h.sum(axis=1), d.n - steps)
        assert e == cl.size


def test_edge_cases(pkg, oracle):
    # paper's 5-node example realised by an edge list, isolated nodes, empty graph
    import torch
    seqs = ["CASSF"] * 7
    res, lens = from_strings(seqs)
    with pkg.TcrNet(0) as net:
        net.load(res, lens)
        with pytest.raises(pkg.TcrNetError) as ei:
            net.components()
        assert ei.value.status == pkg.ERR_STATE
        pairs = np.array([[0, 1], [0, 2], [1, 4], [3, 4]], dtype=np.int64)  # nodes 5, 6 isolated
        net.assemble(torch.from_numpy((pairs[:, 0] << 32) | pairs[:, 1]).cuda())
        row_ptr, col, deg = oracle.csr(pairs, 7)
        check_all_observables(net, oracle, row_ptr, col, deg, seed=1)
        label, size, ncomp, lcc = net.components()
        assert label.tolist() == [0, 0, 0, 0, 0, 5, 6] and size.tolist() == [5] * 5 + [1, 1] and (ncomp, lcc) == (3, 5)
        assert net.neighbor_degree()[2].tolist() == [0.0, 2.0, 10 / 6]
        # removal order errors
        for bad in ([0, 1, 2, 3, 4, 5, 5], [0, 1, 2, 3, 4, 5, 7], [-1, 1, 2, 3, 4, 5, 6]):
            with pytest.raises(pkg.TcrNetError) as ei:
                net.percolation(np.array(bad, dtype=np.int32), [0])
            assert ei.value.status == pkg.ERR_ARG
        with pytest.raises(pkg.TcrNetError):
            net.percolation(np.arange(7, dtype=np.int32), [8])
        out = net.percolation(np.arange(7, dtype=np.int32), [])
        assert out[0].size == 0
        # empty graph
        net.assemble(torch.empty(0, dtype=torch.int64, device="cuda"))
        check_all_observables(net, oracle, *oracle.csr(np.zeros((0, 2), dtype=np.int64), 7), seed=2)
        # the complete graph by a real build: observables follow the CSR of the latest build / restrict
        net.build(0)
        assert net.components()[2:] == (1, 7) and net.degree_histogram().tolist() == [0] * 6 + [7]
    res1, lens1 = from_strings(["CAF"])
    with pkg.TcrNet(0) as net:
        net.load(res1, lens1)
        net.build(1)
        assert net.components()[2:] == (1, 1) and net.degree_histogram().tolist() == [1]
        lcc, n1, n2, h = net.percolation([0], [0, 1], deg_hist=True)
        assert lcc.tolist() == [1, 0] and n1.tolist() == [1.0, 0.0] and n2.tolist() == [1.0, 0.0]


def test_observables_follow_restrict(pkg, oracle):
    """LCC as a function of l_max from ONE build (Fig. 2(i)): restrict, then components."""
    d = generate("cfg1")
    with pkg.TcrNet(0) as net:
        net.load(d.residues, d.lengths)
        net.build(4)
        seen = []
        for l in (4, 3, 2, 1, 0):
            net.restrict(l)
            row_ptr, col, deg, _ = oracle.network(d.residues, d.lengths, l, tier=1)
            _, _, o_ncomp, o_lcc = oracle.components(row_ptr, col)
            assert net.components()[2:] == (o_ncomp, o_lcc)
            assert np.array_equal(net.degree_histogram().cpu().numpy(), oracle.degree_histogram(deg))
            seen.append(o_lcc)
        assert seen == sorted(seen, reverse=True)
