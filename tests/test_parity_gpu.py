"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bar: bit-exact (integer / index work; the result is unique).  Configs 1-4 are compared in full
(element by element, or - configs 3 and 4 - through SHA-256 digests of the whole network that the
oracle-only script tests/golden/make_config_hashes.py wrote); config 5 on the full neighbourhoods of
2,000 uniformly drawn nodes, on every emitted edge, and on properties that hold at any size.
"""
import itertools

import numpy as np
import pytest

from cdr3_synth import generate
from cdr3_synth.generator import from_strings
from helpers import assert_same_network, check_csr_invariants

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


def gpu_network(pkg, residues, lengths, l_max, opts=None):
    with pkg.TcrNet(0) as net:
        for k, v in (opts or {}).items():
            net.set_option(k, v)
        net.load(residues, lengths)
        net.build(l_max)
        out = net.copy_csr()
        out_stats = net.get_stats()
    return out, out_stats


# ------------------------------------------------------------------ full comparisons
@pytest.mark.parametrize("l_max", [0, 1, 2, 3, 5])
def test_cfg1_full(pkg, oracle, l_max):
    d = generate("cfg1")
    got, st = gpu_network(pkg, d.residues, d.lengths, l_max)
    want = oracle.network(d.residues, d.lengths, l_max, tier=0)[:3]
    assert_same_network(got, want)
    check_csr_invariants(*got, d.n)
    assert st["pairs_all"] == d.n * (d.n - 1) // 2 and st["launches_build"] > 0
    # TCRNET_OPT_TIMING: 2 = an event around every phase (the build then runs its phases one after the other, each behind
    # its own read-back), 0 = none; the default 1 launches step A6 behind the distance kernels on the device's edge count
    for level in (2, 0):
        got2, st2 = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_TIMING: level})
        assert_same_network(got2, want)
        assert (st2["ms_build"] > 0) == (level == 2) and (st2["ms_kernel"] > 0) == (level == 2)


@pytest.mark.parametrize("l_max,tier", [(1, 1), (2, 0)])
def test_cfg2_full(pkg, oracle, l_max, tier):
    """N = 50,000: several hundred tiles, ragged tails in every bucket."""
    d = generate("cfg2")
    got, st = gpu_network(pkg, d.residues, d.lengths, l_max)
    want = oracle.network(d.residues, d.lengths, l_max, tier=tier)[:3]
    assert_same_network(got, want)
    check_csr_invariants(*got, d.n)


def test_early_exit_and_schedule_do_not_change_the_result(pkg):
    """the abort only saves time.  Every test position, early exit off, small
    text chunks and a tiny edge buffer (forces the second distance pass) give the same bytes."""
    d = generate("cfg2", n=20000)
    for l_max in (1, 3):
        ref, st0 = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_EARLY_EXIT: 0})
        assert st0["first_check"] == 0
        for fc in range(3, 9):
            got, st = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_FIRST_CHECK: fc})
            assert st["first_check"] == fc
            assert_same_network(got, ref)
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max,
                              {pkg.OPT_TEXT_CHUNK: 256, pkg.OPT_EDGE_CAPACITY: 100, pkg.OPT_DEDUP: 0})
        assert st["distance_passes"] == 2
        assert_same_network(got, ref)
        # collapsed load: the record buffer and / or the expanded edge buffer have to grow
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_EDGE_CAPACITY: 100})
        assert_same_network(got, ref)
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_COUNT_WORK: 1, pkg.OPT_PREFIX_TRIE: 0})
        assert_same_network(got, ref)
        assert 0 < st["lane_columns_exec"] and st["lane_pairs_exec"] >= st["pairs_kept"]
        assert st["work_items_trie"] == 0


def test_prefix_trie_does_not_change_the_result(pkg, oracle):
    """The prefix-trie kernel (TCRNET_OPT_SEGMENT_JOIN = 0) against the text-chunk kernel and the oracle: every first
    test level, tiny trie chunks (chunk borders inside trie nodes), work counters on."""
    d = generate("cfg2", n=20000)
    trie = {pkg.OPT_SEGMENT_JOIN: 0}
    for l_max in (0, 1, 2, 3, 4):
        ref, st0 = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_PREFIX_TRIE: 0, **trie})
        assert st0["work_items_trie"] == 0 and st0["join_mode"] == 0
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max, trie)
        assert st["work_items_trie"] > 0 and st["trie_nodes"] > d.n and st["join_mode"] == 0
        assert_same_network(got, ref)
        for ft in range(3, 7):
            got, st = gpu_network(pkg, d.residues, d.lengths, l_max,
                                  {pkg.OPT_FIRST_CHECK: ft, pkg.OPT_TRIE_CHUNK: 256 * ft, pkg.OPT_COUNT_WORK: ft & 1, **trie})
            assert st["first_check"] == ft and st["work_items_trie"] > 0
            assert_same_network(got, ref)
            if ft & 1:
                assert st["lane_prefix_tests_exec"] > 0 and st["lane_columns_exec"] > 0
    want = oracle.network(d.residues, d.lengths, 2, tier=1)[:3]
    got, _ = gpu_network(pkg, d.residues, d.lengths, 2, trie)
    assert_same_network(got, want)


def test_segment_join_does_not_change_the_result(pkg, oracle):
    """The segment join (pigeonhole candidate filter, the default for l_max <= 6) against the oracle and against the
    paths that visit every length-compatible pair: every threshold it serves, collapse on / off, counters on, a tiny
    edge buffer (second pass), and the l_max <= 1 option."""
    d = generate("cfg2", n=20000)
    for l_max in (0, 1, 2, 3, 4, 5, 6):
        want = oracle.network(d.residues, d.lengths, l_max, tier=1)[:3]
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max)
        assert st["join_mode"] >= 1 and st["work_items_join"] > 0 and st["work_items_trie"] == 0
        assert_same_network(got, want)
        for opts in ({pkg.OPT_SEGMENT_JOIN: 1, pkg.OPT_DEDUP: 0}, {pkg.OPT_SEGMENT_JOIN: 1, pkg.OPT_COUNT_WORK: 1},
                     {pkg.OPT_SEGMENT_JOIN: 1, pkg.OPT_EDGE_CAPACITY: 64}, {pkg.OPT_SEGMENT_JOIN: 1, pkg.OPT_DEDUP: 0, pkg.OPT_EDGE_CAPACITY: 64}):
            got, st = gpu_network(pkg, d.residues, d.lengths, l_max, opts)
            assert st["join_mode"] >= 1
            if opts.get(pkg.OPT_COUNT_WORK):
                assert st["join_probes"] > 0 and st["join_entries"] > 0 and (st["join_candidates"] > 0 or l_max == 0)
            if opts.get(pkg.OPT_EDGE_CAPACITY) and opts.get(pkg.OPT_DEDUP) == 0 and l_max > 0:
                # (the record buffer of a collapsed load starts at n_distinct entries; 3: the verification queue of
                # the join grew as well)
                assert st["distance_passes"] in (2, 3)
            assert_same_network(got, want)
        if l_max <= 1:
            got, st = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_FAST_L1: 1})
            assert st["join_mode"] == 2
            assert_same_network(got, want)
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_SEGMENT_JOIN: 0})
        assert st["join_mode"] == 0
        assert_same_network(got, want)
    # beyond the thresholds the join serves, the rectangular mode and early exit off: the other kernels
    got, st = gpu_network(pkg, d.residues, d.lengths, 7)
    assert st["join_mode"] == 0
    got, st = gpu_network(pkg, d.residues, d.lengths, 2, {pkg.OPT_EARLY_EXIT: 0})
    assert st["join_mode"] == 0


def test_segment_cuts_follow_the_residue_statistics(pkg, oracle):
    """Conserved ends (real CDR3-beta: CASS.. / ..EQYF) leave the outer segments of an even cut with one or two
    informative residues; the load samples the residues per position and the index cuts where the least informative
    segment gains most (make_join_tables).  Any cut is exact: the CASS-shaped stress input and an input whose first
    six residues only are conserved (the cut moves at l_max = 1 too), every threshold of the join, against the oracle."""
    d = generate("cfg4_cass", n=12000)
    for l_max in (0, 1, 2, 3, 4):
        want = oracle.network(d.residues, d.lengths, l_max, tier=1)[:3]
        got, st = gpu_network(pkg, d.residues, d.lengths, l_max)
        # (l_max <= 1: the two halves of a text with four conserved residues at either end are balanced as they are)
        assert st["join_mode"] >= 1 and (st["join_adapted_lengths"] > 0 or l_max <= 1)
        assert_same_network(got, want)
        got, _ = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_DEDUP: 0})
        assert_same_network(got, want)
    rng = np.random.default_rng(77)
    letters = "ACDEFGHIKLMNPQRSTVWY"
    strings = []
    for _ in range(1500):
        s0 = list("CASSLG") + [letters[i] for i in rng.integers(0, 20, int(rng.integers(4, 14)))]
        strings.append("".join(s0))
        for _ in range(int(rng.integers(0, 4))):
            t = list(s0)
            for _ in range(int(rng.integers(1, 4))):
                q = int(rng.integers(5, len(t)))
                op = int(rng.integers(0, 3))
                if op == 0:
                    t[q] = letters[int(rng.integers(0, 20))]
                elif op == 1:
                    t.insert(q, letters[int(rng.integers(0, 20))])
                elif len(t) > 8:
                    del t[q]
            strings.append("".join(t))
    res, ln = from_strings([strings[i] for i in rng.permutation(len(strings))])
    for l_max in (1, 2, 3, 5, 6):
        want = oracle.network(res, ln, l_max, tier=0)[:3]
        got, st = gpu_network(pkg, res, ln, l_max)
        assert st["join_adapted_lengths"] > 0
        assert_same_network(got, want)
    # a load whose positions are all equally informative keeps the even cut
    _, st = gpu_network(pkg, *[getattr(generate("cfg2", n=20000), k) for k in ("residues", "lengths")], 2)
    assert st["join_adapted_lengths"] == 0


def test_prefix_trie_shared_prefixes_and_short_buckets(pkg, oracle):
    """Real CDR3-beta rows mostly start CASS...: few distinct prefixes, deep shared runs, many
    duplicates; plus buckets shorter than the trie depth (they take the text-chunk kernel), every
    l_max the trie kernel is specialised on (0..4), and an l_max beyond them (text-chunk kernel only)."""
    rng = np.random.default_rng(23)
    letters = "ACDEFGHIKLMNPQRSTVWY"
    strings = []
    for _ in range(3000):
        length = int(rng.integers(3, 19))
        body = "".join(letters[i] for i in rng.integers(0, 20, max(0, length - 4)))
        s = ("CASS" + body)[:length]
        strings.append(s)
        for _ in range(int(rng.integers(0, 3))):
            t = list(s)
            k = int(rng.integers(0, 3))
            q = int(rng.integers(0, len(t)))
            if k == 0:
                t[q] = letters[int(rng.integers(0, 20))]
            elif k == 1:
                t.insert(q, letters[int(rng.integers(0, 20))])
            elif len(t) > 1:
                del t[q]
            strings.append("".join(t))
    order = rng.permutation(len(strings))
    res, ln = from_strings([strings[i] for i in order])
    for l_max, opts in ((0, {}), (1, {}), (2, {}), (3, {pkg.OPT_TRIE_CHUNK: 256}), (4, {}), (4, {pkg.OPT_TRIE_CHUNK: 512}),
                        (6, {pkg.OPT_FIRST_CHECK: 3}), (7, {})):
        want = oracle.network(res, ln, l_max, tier=0)[:3]
        got, st = gpu_network(pkg, res, ln, l_max, {pkg.OPT_SEGMENT_JOIN: 0, **opts})
        assert (st["work_items_trie"] > 0) == (l_max <= 4) and st["join_mode"] == 0
        assert_same_network(got, want)
        # the default path: the segment join for the buckets long enough to be cut into l_max + 1 segments, the
        # text-chunk kernel for the shorter ones (lengths 3..19 here: both occur for l_max >= 3)
        got, st = gpu_network(pkg, res, ln, l_max, opts)
        assert (st["join_mode"] >= 1) == (l_max <= 6)
        assert_same_network(got, want)
        if l_max <= 1:
            got, st = gpu_network(pkg, res, ln, l_max, {pkg.OPT_FAST_L1: 1})
            assert_same_network(got, want)


def test_device_load_equals_host_load(pkg):
    import torch
    d = generate("cfg1")
    ref, _ = gpu_network(pkg, d.residues, d.lengths, 2)
    with pkg.TcrNet(0) as net:
        net.load(torch.from_numpy(d.residues).cuda(), torch.from_numpy(d.lengths).cuda())
        net.build(2)
        rp, cl = net.csr()
        dg = net.degrees()
        got = (rp.cpu().numpy(), cl.cpu().numpy(), dg.cpu().numpy())
        assert_same_network(got, ref)
        # repeated builds on one load, different thresholds
        e1 = net.build(1)
        e3 = net.build(3)
        assert e1 <= int(ref[0][-1]) <= e3


# ------------------------------------------------------------------ edge cases
def test_single_and_pair(pkg):
    got, _ = gpu_network(pkg, *from_strings(["CASSF"]), 3)
    assert got[0].tolist() == [0, 0] and got[1].size == 0 and got[2].tolist() == [0]
    got, _ = gpu_network(pkg, *from_strings(["CASSF", "CASSF"]), 0)
    assert got[0].tolist() == [0, 1, 1] and got[1].tolist() == [1] and got[2].tolist() == [1, 1]
    got, _ = gpu_network(pkg, *from_strings(["CASSF", "CASTF"]), 0)
    assert got[1].size == 0
    got, _ = gpu_network(pkg, *from_strings(["CASSF", "CASTF"]), 1)
    assert got[1].tolist() == [1]


def test_paper_five_node_example(pkg):
    """PAPER.md:305-318 realised by strings at l_max = 1 (see tests/golden/paper_adjacency_example.txt)."""
    got, _ = gpu_network(pkg, *from_strings(["AAAA", "AAAB", "AACA", "AEDB", "AADB"]), 1)
    assert got[0].tolist() == [0, 2, 3, 3, 4, 4] and got[1].tolist() == [1, 2, 4, 4] and got[2].tolist() == [2, 2, 1, 1, 2]


def test_all_duplicates_complete_graph(pkg, oracle):
    """Reading Q3: r copies -> K_r for every l_max; r chosen to leave ragged warps and tiles."""
    r = 777
    res, ln = from_strings(["CASSLGQGNTEAFF"] * r)
    for l_max in (0, 2):
        got, _ = gpu_network(pkg, res, ln, l_max)
        assert int(got[0][-1]) == r * (r - 1) // 2
        assert (got[2] == r - 1).all()
        check_csr_invariants(*got, r)


@pytest.mark.parametrize("l_max", [0, 1, 3])
def test_collapsing_identical_sequences_does_not_change_the_result(pkg, oracle, l_max):
    """TCRNET_OPT_DEDUP: the distance step over the distinct sequences + multiplied emission (groups of 1, 2, many
    rows on either side, cliques inside a group) equals the row-by-row build and the oracle."""
    d = generate("cfg1")
    on, st_on = gpu_network(pkg, d.residues, d.lengths, l_max)
    off, st_off = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_DEDUP: 0})
    assert st_on["n_distinct"] < d.n == st_off["n_distinct"]
    assert st_on["n_distinct"] == len({bytes(r) for r in np.split(d.residues, np.cumsum(d.lengths)[:-1])})
    assert st_on["pairs_kept"] < st_off["pairs_kept"] and st_on["pairs_all"] == st_off["pairs_all"]
    assert_same_network(on, off)
    assert_same_network(on, oracle.network(d.residues, d.lengths, l_max, tier=0)[:3])
    # hubs: two sequences at distance 1 with many rows each, next to singletons and a third shared sequence
    strings = ["CASSLGQF"] * 70 + ["CASSLGQW"] * 45 + ["CASSLGQ", "CASSLGQFF", "CWWWW"] + ["CASRLGQF"] * 3
    rng = np.random.default_rng(5)
    strings = [strings[i] for i in rng.permutation(len(strings))]
    res, ln = from_strings(strings)
    got, st = gpu_network(pkg, res, ln, l_max)
    assert st["n_distinct"] == 6
    assert_same_network(got, oracle.network(res, ln, l_max, tier=0)[:3])


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_heavily_repeated_rows_random(pkg, oracle, seed):
    """Random multiplicities (1 .. 60 rows per sequence) over a family-structured base set, shuffled; every l_max,
    also with an edge buffer that has to grow (records and expansion)."""
    rng = np.random.default_rng(100 + seed)
    d = generate("cfg1", n=400)
    rows = np.split(d.residues, np.cumsum(d.lengths)[:-1])
    mult = rng.choice([1, 1, 1, 2, 3, 7, 25, 60], size=len(rows))
    strings = [bytes(rows[i]).decode() for i in range(len(rows)) for _ in range(int(mult[i]))]
    strings = [strings[i] for i in rng.permutation(len(strings))]
    res, ln = from_strings(strings)
    for l_max in (0, 1, 2):
        want = oracle.network(res, ln, l_max, tier=1)[:3]
        got, st = gpu_network(pkg, res, ln, l_max)
        assert st["n_distinct"] == len(set(strings))
        assert_same_network(got, want)
        got, _ = gpu_network(pkg, res, ln, l_max, {pkg.OPT_EDGE_CAPACITY: 7})
        assert_same_network(got, want)
    check_csr_invariants(*got, len(strings))


def test_products_of_two_heavily_repeated_sequences(pkg, oracle):
    """Two neighbouring sequences that many rows share: rows x rows edges from ONE recorded pair (90 x 70, 200 x 90,
    beyond what one warp expands itself: the product is spread over the grid), next to ordinary rows; every threshold,
    also with buffers that have to grow."""
    rng = np.random.default_rng(77)
    d = generate("cfg1", n=300)
    base = [bytes(r).decode() for r in np.split(d.residues, np.cumsum(d.lengths)[:-1])]
    strings = base + ["CASSLGQYF"] * 90 + ["CASSLGEYF"] * 70 + ["CASSLEYF"] * 200 + ["CASSLGQAYF"] * 3
    strings = [strings[i] for i in rng.permutation(len(strings))]
    res, ln = from_strings(strings)
    for l_max in (1, 2):
        want = oracle.network(res, ln, l_max, tier=0)[:3]
        for opts in ({}, {pkg.OPT_EDGE_CAPACITY: 50}, {pkg.OPT_SEGMENT_JOIN: 0}, {pkg.OPT_DEDUP: 0}):
            got, st = gpu_network(pkg, res, ln, l_max, opts)
            assert_same_network(got, want)
    assert int(want[0][-1]) > 90 * 70 + 200 * 90


def test_rows_of_every_sorting_regime(pkg, oracle):
    """The CSR step orders a row by ranking (<= 256 neighbours, one thread per edge), by a bitonic network in shared
    memory (<= 8192) or in place (beyond): a clique of 9,001 copies has rows of every such length; the other strings
    hang off it."""
    strings = ["CASSLGQF"] * 5000 + ["CASSLGQW", "CASRLGQF", "CWWWWWWW"] + ["CASSLGQF"] * 4001 + ["CASSLGF"] * 40
    res, ln = from_strings(strings)
    got, _ = gpu_network(pkg, res, ln, 1)
    want = oracle.network(res, ln, 1, tier=1)[:3]
    assert_same_network(got, want)
    check_csr_invariants(*got, len(strings))
    assert int(np.diff(got[0]).max()) > 8192


def test_lmax_at_least_max_length_gives_complete_graph(pkg, oracle):
    d = generate("cfg1", n=300)
    got, _ = gpu_network(pkg, d.residues, d.lengths, 25)
    assert int(got[0][-1]) == 300 * 299 // 2
    got, _ = gpu_network(pkg, d.residues, d.lengths, 64)
    assert int(got[0][-1]) == 300 * 299 // 2


def test_all_lengths_1_to_64_incl_wide_words(pkg, oracle):
    """Lengths 1..64 (patterns > 32 take the 64-bit kernel), tiny alphabet so that edges exist,
    several thresholds incl. ones larger than the first-test column."""
    rng = np.random.default_rng(11)
    strings = []
    for length in range(1, 65):
        base = "".join("ACD"[i] for i in rng.integers(0, 3, length))
        strings.append(base)
        for _ in range(6):
            s = list(base)
            for _ in range(int(rng.integers(0, 4))):
                k = int(rng.integers(0, 3))
                p = int(rng.integers(0, len(s)))
                if k == 0:
                    s[p] = "ACD"[int(rng.integers(0, 3))]
                elif k == 1 and len(s) < 64:
                    s.insert(p, "ACD"[int(rng.integers(0, 3))])
                elif k == 2 and len(s) > 1:
                    del s[p]
            strings.append("".join(s))
    order = rng.permutation(len(strings))
    strings = [strings[i] for i in order]
    res, ln = from_strings(strings)
    for l_max in (0, 1, 2, 4, 9, 20):
        got, _ = gpu_network(pkg, res, ln, l_max)
        want = oracle.network(res, ln, l_max, tier=0)[:3]
        assert_same_network(got, want)
        got, _ = gpu_network(pkg, res, ln, l_max, {pkg.OPT_EARLY_EXIT: 0})
        assert_same_network(got, want)


@pytest.mark.parametrize("alphabet,lo,hi", [("AC", 4, 22), ("AIQY", 6, 40), ("ABCDEFGHIJKLMNOPQRSTUVWXYZ", 30, 64), ("A", 1, 64)])
def test_low_complexity_sequences(pkg, oracle, alphabet, lo, hi):
    """Repetitive strings over tiny alphabets (many diagonals match at once, the composition counts saturate, residues
    of one class - A, I, Q, Y share code & 7 - and segments repeat inside a string), random strings over all 26 letters
    up to 64 residues (64-bit planes), and runs of one letter: every threshold the join serves + one beyond it, against
    the tier-0 oracle."""
    rng = np.random.default_rng(len(alphabet) * 1000 + hi)
    strings = []
    for _ in range(500):
        n = int(rng.integers(lo, hi + 1))
        s = "".join(alphabet[i] for i in rng.integers(0, len(alphabet), n))
        strings.append(s)
        for _ in range(int(rng.integers(0, 4))):  # a few neighbours: up to 3 random edits
            t = list(s)
            for _ in range(int(rng.integers(1, 4))):
                k = int(rng.integers(0, 3))
                q = int(rng.integers(0, len(t)))
                c = alphabet[int(rng.integers(0, len(alphabet)))]
                if k == 0:
                    t[q] = c
                elif k == 1 and len(t) < 64:
                    t.insert(q, c)
                elif k == 2 and len(t) > 1:
                    del t[q]
            strings.append("".join(t))
    strings = [strings[i] for i in rng.permutation(len(strings))]
    res, ln = from_strings(strings)
    for l_max in (0, 1, 2, 3, 4, 5, 6, 7):
        want = oracle.network(res, ln, l_max, tier=0)[:3]
        got, st = gpu_network(pkg, res, ln, l_max)
        assert st["join_mode"] == 0 if l_max > 6 else (st["join_mode"] >= 1 or st["pairs_kept"] == 0)
        assert_same_network(got, want)
        if l_max in (1, 3):
            got, _ = gpu_network(pkg, res, ln, l_max, {pkg.OPT_DEDUP: 0})
            assert_same_network(got, want)


@pytest.mark.parametrize("seed", range(6))
def test_many_small_random_instances(pkg, oracle, seed):
    """Forty small random inputs per seed - short strings (1..14 residues: segments of one residue, texts barely long
    enough to be cut into l_max + 1 segments, buckets that stay with the text-chunk kernel), alphabets of 2..6 letters
    (dense networks, many pairs found through several probes), a third of the rows repeated - at every threshold 0..5,
    collapse on and off, against the tier-0 oracle."""
    rng = np.random.default_rng(9000 + seed)
    letters = "ACDEFGHIKLMNPQRSTVWY"
    with pkg.TcrNet(0) as net, pkg.TcrNet(0) as net_rows:
        net_rows.set_option(pkg.OPT_DEDUP, 0)
        for _ in range(40):
            k = int(rng.integers(2, 7))
            alpha = [letters[i] for i in rng.choice(20, k, replace=False)]
            lo = int(rng.integers(1, 6))
            hi = lo + int(rng.integers(0, 10))
            n = int(rng.integers(2, 180))
            strings = ["".join(alpha[i] for i in rng.integers(0, k, int(rng.integers(lo, hi + 1)))) for _ in range(n)]
            strings += [strings[i] for i in rng.integers(0, n, n // 3)]
            res, ln = from_strings(strings)
            for l_max in range(8):
                want = oracle.network(res, ln, l_max, tier=0)[:3]
                for ctx in (net, net_rows):
                    ctx.load(res, ln)
                    ctx.build(l_max)
                    assert_same_network(ctx.copy_csr(), want)


@pytest.mark.parametrize("seed", range(3))
def test_many_small_random_instances_long_rows(pkg, oracle, seed):
    """The same with rows of 20..64 residues (64-bit planes as soon as one row exceeds 32; pairs whose text is longer
    than 32 while the pattern is not) and planted neighbours (1..5 random edits of an earlier row)."""
    rng = np.random.default_rng(9100 + seed)
    letters = "ACDEFGHIKLMNPQRSTVWY"
    with pkg.TcrNet(0) as net:
        for _ in range(25):
            k = int(rng.integers(3, 21))
            lo = int(rng.integers(20, 40))
            hi = min(64, lo + int(rng.integers(0, 30)))
            strings = []
            for _ in range(int(rng.integers(5, 60))):
                s0 = [letters[i] for i in rng.integers(0, k, int(rng.integers(lo, hi + 1)))]
                strings.append("".join(s0))
                for _ in range(int(rng.integers(0, 4))):
                    t = list(s0)
                    for _ in range(int(rng.integers(1, 6))):
                        q = int(rng.integers(0, len(t)))
                        op = int(rng.integers(0, 3))
                        if op == 0:
                            t[q] = letters[int(rng.integers(0, k))]
                        elif op == 1 and len(t) < 64:
                            t.insert(q, letters[int(rng.integers(0, k))])
                        elif op == 2 and len(t) > 1:
                            del t[q]
                    strings.append("".join(t))
            res, ln = from_strings(strings)
            for l_max in range(8):
                want = oracle.network(res, ln, l_max, tier=0)[:3]
                net.load(res, ln)
                net.build(l_max)
                assert_same_network(net.copy_csr(), want)


@pytest.mark.parametrize("seed", range(3))
def test_many_small_random_instances_cdr3_families(pkg, oracle, seed):
    """The same with CDR3-shaped rows: conserved first / last residue, 8..25 residues, families of a seed and up to
    seven copies with 0..4 random edits each, a third of all rows repeated, shuffled."""
    rng = np.random.default_rng(9200 + seed)
    letters = "ACDEFGHIKLMNPQRSTVWY"
    with pkg.TcrNet(0) as net, pkg.TcrNet(0) as net_rows:
        net_rows.set_option(pkg.OPT_DEDUP, 0)
        for _ in range(30):
            strings = []
            for _ in range(int(rng.integers(5, 120))):
                s0 = ["C"] + [letters[i] for i in rng.integers(0, 20, int(rng.integers(6, 24)))] + ["F"]
                strings.append("".join(s0))
                for _ in range(int(rng.integers(0, 8))):
                    t = list(s0)
                    for _ in range(int(rng.integers(0, 5))):
                        q = int(rng.integers(0, len(t)))
                        op = int(rng.integers(0, 3))
                        if op == 0:
                            t[q] = letters[int(rng.integers(0, 20))]
                        elif op == 1:
                            t.insert(q, letters[int(rng.integers(0, 20))])
                        elif len(t) > 2:
                            del t[q]
                    strings.append("".join(t))
            strings += [strings[i] for i in rng.integers(0, len(strings), len(strings) // 3)]
            strings = [strings[i] for i in rng.permutation(len(strings))]
            res, ln = from_strings(strings)
            for l_max in range(8):
                want = oracle.network(res, ln, l_max, tier=0)[:3]
                for ctx in (net, net_rows):
                    ctx.load(res, ln)
                    ctx.build(l_max)
                    assert_same_network(ctx.copy_csr(), want)


def test_length_64_and_all_26_letters(pkg, oracle):
    rng = np.random.default_rng(5)
    letters = "ABCDEFGHIJKLMNOPQRSTUVWXYZ"
    strings = []
    for _ in range(40):
        base = [letters[i] for i in rng.integers(0, 26, 64)]
        strings.append("".join(base))
        for k in range(1, 4):
            s = base[:]
            for p in rng.choice(64, k, replace=False):
                s[p] = letters[int(rng.integers(0, 26))]
            strings.append("".join(s))
            strings.append("".join(s[1:]))  # one deletion at the front: length 63
    res, ln = from_strings(strings)
    for l_max in (1, 3):
        got, _ = gpu_network(pkg, res, ln, l_max)
        assert_same_network(got, oracle.network(res, ln, l_max, tier=0)[:3])


def test_equal_length_is_not_hamming(pkg):
    """Reading Q6: a cyclic shift has Hamming distance 4 but Levenshtein distance 2."""
    got, _ = gpu_network(pkg, *from_strings(["ABCD", "BCDA"]), 2)
    assert got[1].tolist() == [1]
    got, _ = gpu_network(pkg, *from_strings(["ABCD", "BCDA"]), 1)
    assert got[1].size == 0


def test_errors(pkg):
    with pkg.TcrNet(0) as net:
        with pytest.raises(pkg.TcrNetError) as e:
            net.build(1)
        assert e.value.status == pkg.ERR_STATE
        for bad in (0, 65):
            with pytest.raises(pkg.TcrNetError) as e:
                net.load(np.full(70, ord("A"), np.uint8), np.array([5, bad], np.int32))
            assert e.value.status == pkg.ERR_LENGTH
        with pytest.raises(pkg.TcrNetError) as e:
            net.load(np.frombuffer(b"CASSaF", np.uint8), np.array([6], np.int32))
        assert e.value.status == pkg.ERR_RESIDUE
        with pytest.raises(pkg.TcrNetError) as e:
            net.csr()
        assert e.value.status == pkg.ERR_STATE
        res, ln = from_strings(["CASSF"] * 50)
        net.load(res, ln)
        for bad in (-1, 65):
            with pytest.raises(pkg.TcrNetError) as e:
                net.build(bad)
            assert e.value.status == pkg.ERR_LMAX
        net.set_option(pkg.OPT_EDGE_LIMIT, 100)
        with pytest.raises(pkg.TcrNetError) as e:
            net.build(0)  # 1225 edges > limit
        assert e.value.status == pkg.ERR_EDGE_OVERFLOW
        net.set_option(pkg.OPT_EDGE_LIMIT, 1 << 31)
        assert net.build(0) == 1225  # the context stays usable
        with pytest.raises(pkg.TcrNetError):
            net.set_option(99, 1)


def test_one_heavily_repeated_sequence_fails_fast(pkg):
    """70,000 identical rows would be 2.45e9 clique edges, more than the hard limit of 2^31: the build refuses at once
    (the count is known at load) instead of enumerating them; with a limit that admits them a smaller clique is built."""
    import time
    rows = ["CASSLGQYF"] * 70000 + ["CASSLGEYF", "CAWSVGF"]
    res, ln = from_strings(rows)
    with pkg.TcrNet(0) as net:
        net.load(res, ln)
        t0 = time.perf_counter()
        with pytest.raises(pkg.TcrNetError) as e:
            net.build(1)
        assert e.value.status == pkg.ERR_EDGE_OVERFLOW and time.perf_counter() - t0 < 0.5
        res2, ln2 = from_strings(["CASSLGQYF"] * 3000 + ["CASSLGEYF", "CAWSVGF"])
        net.load(res2, ln2)
        net.set_option(pkg.OPT_EDGE_LIMIT, 1_000_000)
        with pytest.raises(pkg.TcrNetError) as e:
            net.build(0)
        assert e.value.status == pkg.ERR_EDGE_OVERFLOW
        net.set_option(pkg.OPT_EDGE_LIMIT, 1 << 31)
        assert net.build(1) == 3000 * 2999 // 2 + 3000
        rp, cl, dg = net.copy_csr()
        check_csr_invariants(rp, cl, dg, 3002)
        assert dg[:3000].tolist() == [3000] * 3000 and dg[3000] == 3000 and dg[3001] == 0


def test_collapse_pauses_after_a_load_without_repeats(pkg, oracle):
    """A load that finds no repeated sequence hands the offsets / histogram / sort keys it computed on to the pack, and
    the next seven loads of the context do not try to collapse (TCRNET_OPT_DEDUP re-arms it).  None of it changes a
    result: a series of loads with and without repeated rows on ONE context, each against the oracle."""
    d = generate("cfg2", n=20000)
    off = np.concatenate([[0], np.cumsum(d.lengths.astype(np.int64))])
    first = {}
    for i in range(d.n):
        first.setdefault(d.residues[off[i]:off[i + 1]].tobytes(), i)
    keep = np.array(sorted(first.values()))
    assert keep.size < d.n
    u_res = np.concatenate([d.residues[off[i]:off[i + 1]] for i in keep])
    u_len = np.ascontiguousarray(d.lengths[keep])
    want_u = {l_max: oracle.network(u_res, u_len, l_max, tier=1)[:3] for l_max in (1, 2)}
    want_d = {l_max: oracle.network(d.residues, d.lengths, l_max, tier=1)[:3] for l_max in (1, 2)}
    with pkg.TcrNet(0) as net:
        seen = []
        for k in range(11):
            dup = k in (0, 3, 10)
            if k == 10:
                net.set_option(pkg.OPT_DEDUP, 1)  # re-armed
            net.load(*((d.residues, d.lengths) if dup else (u_res, u_len)))
            for l_max in (1, 2):
                net.build(l_max)
                assert_same_network(net.copy_csr(), (want_d if dup else want_u)[l_max])
            seen.append(int(net.get_stats()["n_distinct"]))
        n_d, n_u = d.n, int(keep.size)
        # 0: collapsed; 1: attempt, nothing found; 2..8: paused (3: repeated rows go uncollapsed); 9: attempt again;
        # 10: re-armed by the option, collapsed
        assert seen[0] == n_u and seen[1] == n_u and seen[3] == n_d and seen[10] == n_u
        assert all(x == n_u for k, x in enumerate(seen) if k not in (3,))


def test_device_side_validation(pkg):
    import torch
    with pkg.TcrNet(0) as net:
        res = torch.full((20,), ord("A"), dtype=torch.uint8, device="cuda")
        with pytest.raises(pkg.TcrNetError) as e:
            net.load(res, torch.tensor([20, 0], dtype=torch.int32, device="cuda"))
        assert e.value.status == pkg.ERR_LENGTH
        res[7] = ord("~")
        with pytest.raises(pkg.TcrNetError) as e:
            net.load(res, torch.tensor([10, 10], dtype=torch.int32, device="cuda"))
        assert e.value.status == pkg.ERR_RESIDUE
        # total_len must equal sum(lengths), with or without repeated rows, collapse on or off (a residue buffer one
        # byte too short / too long; the binding passes residues.numel() as total_len)
        for dedup in (1, 0):
            net.set_option(pkg.OPT_DEDUP, dedup)
            for rows in (["CASSLF", "CASSF", "CASSLF", "CASSLF", "CAF"], ["CASSLF", "CASSF", "CAWF"]):
                r, ln = from_strings(rows)
                r_d, ln_d = torch.from_numpy(r).cuda(), torch.from_numpy(ln).cuda()
                net.load(r_d, ln_d)
                for bad in (r_d[:-1], torch.cat([r_d, r_d[:1]])):
                    with pytest.raises(pkg.TcrNetError) as e:
                        net.load(bad, ln_d)
                    assert e.value.status == pkg.ERR_ARG


def test_host_loads_reuse_the_buffers_of_the_previous_load(pkg):
    """tcrnet_load[_sized] copies the residues block by block while it sums the lengths whenever the buffer left by the
    previous load is large enough: a small load, a larger one (the buffer grows), the same again (copied in several
    blocks: N > 65,536 rows), a smaller one - each equal to the network of a fresh context.  A residue array shorter
    than sum(lengths) is refused without being read past its end; the four-argument tcrnet_load gives the same."""
    import ctypes as C
    small, large = generate("cfg1"), generate("cfg3")
    want = {id(d): gpu_network(pkg, d.residues, d.lengths, 1)[0] for d in (small, large)}
    with pkg.TcrNet(0) as net:
        for d in (small, large, large, small, large):
            net.load(d.residues, d.lengths)
            net.build(1)
            assert_same_network(net.copy_csr(), want[id(d)])
            with pytest.raises(pkg.TcrNetError) as e:
                net.load(d.residues[:-1], d.lengths)
            assert e.value.status == pkg.ERR_ARG
        r = np.ascontiguousarray(large.residues)
        ln = np.ascontiguousarray(large.lengths)
        rc = net._lib.tcrnet_load(net._ctx, r.ctypes.data_as(C.POINTER(C.c_uint8)),
                                  ln.ctypes.data_as(C.POINTER(C.c_int32)), int(ln.size))
        assert rc == pkg.OK
        net.n = int(ln.size)
        net.build(1)
        assert_same_network(net.copy_csr(), want[id(large)])
        bad = ln.copy()
        bad[150_000] = 65
        with pytest.raises(pkg.TcrNetError) as e:
            net.load(r, bad)
        assert e.value.status == pkg.ERR_LENGTH


# ------------------------------------------------------------------ BASELINE.json's large configs
def _sampled_parity(pkg, oracle, name, l_max, n_sample, seed, opts=None, n=None):
    """What the oracle cannot compute in full: (i) the FULL neighbourhoods of n_sample uniformly drawn nodes (drawn from
    the generator's row count alone, never from the GPU's output) against the tier-1 oracle, every partner visited;
    (ii) EVERY edge the GPU emitted has oracle distance <= l_max (no spurious edge anywhere in the network);
    (iii) CSR invariants; (iv) the generator-linked lower bound over all family pairs."""
    d = generate(name) if n is None else generate(name, n=n)
    (rp, cl, dg), st = gpu_network(pkg, d.residues, d.lengths, l_max, opts)
    check_csr_invariants(rp, cl, dg, d.n)
    rng = np.random.default_rng(seed)
    nodes = np.sort(rng.choice(d.n, n_sample, replace=False))
    pairs, _ = oracle.edges(d.residues, d.lengths, l_max, rows=nodes, all_partners=True, tier=1)
    order = np.argsort(pairs[:, 0], kind="stable")
    pairs = pairs[order]
    cuts = np.searchsorted(pairs[:, 0], nodes, side="left"), np.searchsorted(pairs[:, 0], nodes, side="right")
    # the GPU's neighbourhoods of the sampled nodes: upper part from the node's own row, lower part from the rows
    # that list the node as a column
    rows_of = np.repeat(np.arange(d.n, dtype=np.int64), np.diff(rp))
    hit = np.nonzero(np.isin(cl, nodes))[0]
    lower_of = {}
    for e in hit:
        lower_of.setdefault(int(cl[e]), []).append(int(rows_of[e]))
    n_edges_seen = 0
    for k, u in enumerate(nodes):
        want = np.sort(pairs[cuts[0][k]:cuts[1][k], 1])
        got = np.sort(np.concatenate([np.array(lower_of.get(int(u), []), dtype=np.int64),
                                      cl[rp[u]:rp[u + 1]].astype(np.int64)]))
        assert np.array_equal(got, want), f"node {u}"
        assert dg[u] == want.size
        n_edges_seen += want.size
    assert n_edges_seen > 0
    # (ii) no spurious edge: the oracle's distance of every emitted pair
    all_pairs = np.stack([rows_of, cl.astype(np.int64)], axis=1)
    dist = oracle.lev_pairs(d.residues, d.lengths, all_pairs)
    assert int(dist.max(initial=0)) <= l_max, f"{int((dist > l_max).sum())} emitted edges are farther apart than l_max"
    # (iv) generator-linked lower bound over ALL family pairs: edits sum <= l_max  =>  edge
    order = np.argsort(d.family, kind="stable")
    fam = d.family[order]
    starts = np.nonzero(np.diff(fam, prepend=-2))[0]
    edge_keys = rows_of * d.n + cl
    must = []
    for a, b in zip(starts, list(starts[1:]) + [fam.size]):
        if fam[a] < 0:
            continue
        members = order[a:b]
        low = members[d.n_edits[members] <= l_max]
        for x, y in itertools.combinations(low.tolist(), 2):
            if d.n_edits[x] + d.n_edits[y] <= l_max:
                must.append(min(x, y) * d.n + max(x, y))
        if len(must) > 400000:
            break
    must = np.array(must, dtype=np.int64)
    assert must.size > 0 and np.isin(must, edge_keys).all()
    return st, (rp, cl, dg)


def _golden_digests(name, l_max):
    """tests/golden/<name>_l<l_max>_network.sha256, written by tests/golden/make_config_hashes.py from the oracle alone."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"{name}_l{l_max}_network.sha256")
    if not os.path.exists(path):
        return None
    out = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = v
    return out


@pytest.mark.parametrize("name,l_max", [("cfg1", 1), ("cfg3", 2), ("cfg4", 1)])
def test_whole_network_equals_the_oracles_digest(pkg, name, l_max):
    """The WHOLE network of the config (default launch configuration, what bench.py times) against the tier-1 oracle's
    network: SHA-256 of the exact bytes tcrnet_copy_csr hands back (row_ptr, col, deg) equal the stored digests the
    oracle-only script wrote.  PAPER.md:297 (edge rule), 301-318 (adjacency), 224 (degrees)."""
    import hashlib
    want = _golden_digests(name, l_max)
    assert want is not None, "run tests/golden/make_config_hashes.py"
    d = generate(name)
    assert hashlib.sha256(d.residues.tobytes() + d.lengths.astype("<i4").tobytes()).hexdigest() == want["sha256_input"]
    (rp, cl, dg), st = gpu_network(pkg, d.residues, d.lengths, l_max)
    assert int(rp[-1]) == int(want["n_edges"]) and int(dg.max()) == int(want["max_degree"])
    assert int((dg == 0).sum()) == int(want["n_isolated"])
    b_rp, b_cl, b_dg = (np.ascontiguousarray(rp, dtype="<i8").tobytes(), np.ascontiguousarray(cl, dtype="<i4").tobytes(),
                        np.ascontiguousarray(dg, dtype="<i4").tobytes())
    assert hashlib.sha256(b_rp).hexdigest() == want["sha256_row_ptr"]
    assert hashlib.sha256(b_cl).hexdigest() == want["sha256_col"]
    assert hashlib.sha256(b_dg).hexdigest() == want["sha256_deg"]
    assert hashlib.sha256(b_rp + b_cl + b_dg).hexdigest() == want["sha256_all"]
    if name == "cfg4":
        assert st["pairs_all"] == 800000 * 799999 // 2 and st["distance_passes"] == 1
    # the prefix-trie path gives the same bytes
    (rp2, cl2, dg2), st2 = gpu_network(pkg, d.residues, d.lengths, l_max, {pkg.OPT_SEGMENT_JOIN: 0})
    assert st2["join_mode"] == 0
    assert_same_network((rp2, cl2, dg2), (rp, cl, dg))


def test_cfg3_sampled(pkg, oracle):
    _sampled_parity(pkg, oracle, "cfg3", 2, 2000, 3)


def test_cfg4_sampled_headline_config(pkg, oracle):
    """N = 800,000, l_max = 1: the configuration bench.py times, default launch configuration."""
    st, _ = _sampled_parity(pkg, oracle, "cfg4", 1, 2000, 4)
    assert st["pairs_all"] == 800000 * 799999 // 2
    assert st["distance_passes"] == 1


def test_cfg4_whole_network_is_the_same_row_by_row(pkg):
    """At the full headline size the collapsed build (the default, what bench.py times) equals, byte for byte, the
    build that takes every row as its own pattern / text (two independent paths
    through the kernels; the oracle covers sampled neighbourhoods of the same network in the test above)."""
    d = generate("cfg4")
    on, st_on = gpu_network(pkg, d.residues, d.lengths, 1)
    off, st_off = gpu_network(pkg, d.residues, d.lengths, 1, {pkg.OPT_DEDUP: 0})
    assert st_on["n_distinct"] < st_off["n_distinct"] == d.n
    assert_same_network(on, off)
    check_csr_invariants(*on, d.n)


def test_cass_shaped_input_sampled_at_large_size(pkg, oracle):
    """The stress input of DESIGN.md section 6 (every row CASS...EQYF; here N = 400,000) at l_max = 2, where the segment
    cuts follow the residue statistics: 1,000 uniformly drawn nodes' full neighbourhoods and every one of the 1.9e7
    emitted edges against the oracle."""
    st, _ = _sampled_parity(pkg, oracle, "cfg4_cass", 2, 1000, 6, n=400000)
    assert st["join_mode"] == 1 and st["join_adapted_lengths"] >= 10


def test_cfg5_sampled(pkg, oracle):
    """N = 2,000,000, l_max = 3, length law N(16,3) clipped to [5,40] (the longest row drawn is 30).  The whole network is beyond the oracle
    (about 125 core-hours): 2,000 uniformly drawn nodes' full neighbourhoods, every one of the ~2e7 emitted edges checked
    against the oracle's distance, and the default path byte-equal to the prefix-trie path on a 300,000-row prefix."""
    st, net = _sampled_parity(pkg, oracle, "cfg5", 3, 2000, 5)
    d = generate("cfg5")
    n = 300000
    off = int(d.lengths[:n].astype(np.int64).sum())
    a, _ = gpu_network(pkg, d.residues[:off], d.lengths[:n], 3)
    b, stb = gpu_network(pkg, d.residues[:off], d.lengths[:n], 3, {pkg.OPT_SEGMENT_JOIN: 0})
    assert stb["join_mode"] == 0
    assert_same_network(a, b)


def test_large_n_sort_and_scan_paths(pkg):
    """N = 4,500,000 short rows: beyond the thresholds where the sequence sort switches to 4096-key tiles
    (n >= 4,194,304) and the prefix sums to their three-launch form (n > 2,097,152).  l_max = 0, where the network is
    known without any distance: rows are joined iff their bytes are equal (exact-match join by sorting, the oracle's
    own pin for l_max = 0), so degrees and the edge count follow from the multiplicities.  Both load orders (by length
    only / lexicographic) and both kernels."""
    rng = np.random.default_rng(4500)
    n = 4_500_000
    ln = rng.integers(6, 11, n).astype(np.int32)
    mat = np.frombuffer(b"ACDEFGHIKLMNPQRSTVWY", dtype=np.uint8)[rng.integers(0, 20, (n, 10))]
    mat[np.arange(10)[None, :] >= ln[:, None]] = 0
    res = np.ascontiguousarray(mat[mat != 0])
    _, inv, cnt = np.unique(np.ascontiguousarray(mat).view("V10").ravel(), return_inverse=True, return_counts=True)
    want_deg = (cnt[inv] - 1).astype(np.int32)
    want_edges = int((cnt.astype(np.int64) * (cnt - 1) // 2).sum())
    assert want_edges > 1000
    for opts in ({}, {pkg.OPT_SEGMENT_JOIN: 0}):
        (rp, cl, dg), st = gpu_network(pkg, res, ln, 0, opts)
        # (two different sequences may share a 32-bit fingerprint: the repeated rows of one of them then stay sequences
        # of their own - a few more "distinct" sequences than there are, never a different network)
        assert cnt.size <= st["n_distinct"] <= cnt.size + 100 and int(rp[-1]) == want_edges
        assert np.array_equal(dg, want_deg)
        check_csr_invariants(rp, cl, dg, n)
        rows_of = np.repeat(np.arange(n, dtype=np.int64), np.diff(rp))
        assert np.array_equal(inv[rows_of], inv[cl])  # every edge joins two rows with the same bytes


# ------------------------------------------------------------------ 8(e): shards; 8(f): labels, sweep, query mode
def test_shards_partition_the_edge_set(pkg, oracle):
    """tcrnet_build_shard: the work items are dealt out to the shards interleaved; the shards' key
    lists are disjoint, their union assembled by tcrnet_assemble is the oracle's network."""
    import torch
    d = generate("cfg2", n=20000)
    for l_max, n_shards in ((1, 2), (3, 3), (2, 7)):
        want = oracle.network(d.residues, d.lengths, l_max, tier=1)[:3]
        with pkg.TcrNet(0) as net:
            net.load(d.residues, d.lengths)
            parts = [net.build_shard(l_max, r, n_shards).clone() for r in range(n_shards)]
            allk = torch.cat(parts)
            assert allk.numel() == int(want[0][-1]) and torch.unique(allk).numel() == allk.numel()
            assert sum(p.numel() > 0 for p in parts) == n_shards          # every shard got real work
            assert net.assemble(allk) == int(want[0][-1])
            assert_same_network(net.copy_csr(), want)
            # in-place assemble of one shard's own keys, then a plain build on the same context
            k0 = net.build_shard(l_max, 0, n_shards)
            assert net.assemble(k0) == parts[0].numel()
            rp, cl, dg = net.copy_csr()
            check_csr_invariants(rp, cl, dg, d.n)
            net.build(l_max)
            assert_same_network(net.copy_csr(), want)
            # a key outside the strict upper triangle / the node range is rejected
            bad = allk.clone()
            bad[0] = (5 << 32) | 5
            with pytest.raises(pkg.TcrNetError) as ei:
                net.assemble(bad)
            assert ei.value.status == pkg.ERR_ARG
            bad[0] = (5 << 32) | d.n
            with pytest.raises(pkg.TcrNetError):
                net.assemble(bad)


def test_edge_distances_and_threshold_sweep(pkg, oracle):
    """NEXT-3: labels of a build at l_max = 4 equal the oracle's distances edge by edge, and the
    chain restrict(3), restrict(2), ... reproduces the oracle's network at every threshold
    (Fig. 2(i) sweeps l_max on one repertoire)."""
    d = generate("cfg1")
    off = np.concatenate([[0], np.cumsum(d.lengths)])
    seq = lambda i: d.residues[off[i]:off[i + 1]]
    with pkg.TcrNet(0) as net:
        net.load(d.residues, d.lengths)
        net.build(4)
        rp, cl, dg = net.copy_csr()
        dist = net.edge_distances().cpu().numpy()
        assert dist.shape == cl.shape
        rows = np.repeat(np.arange(d.n), np.diff(rp))
        want_d = np.array([oracle.lev(seq(u), seq(v)) for u, v in zip(rows, cl)], dtype=np.uint8)
        assert np.array_equal(dist, want_d)
        for l in (4, 3, 2, 1, 0):
            e = net.restrict(l)
            want = oracle.network(d.residues, d.lengths, l, tier=0)[:3]
            assert e == int(want[0][-1])
            assert_same_network(net.copy_csr(), want)
            lab = net.edge_distances().cpu().numpy()
            assert lab.size == e and (lab <= l).all()
        with pytest.raises(pkg.TcrNetError) as ei:
            net.restrict(1)      # the network is now the one at l_max = 0
        assert ei.value.status == pkg.ERR_LMAX


def test_edge_distances_long_sequences_and_large_thresholds(pkg, oracle):
    """Labels on 64-bit plane rows (sequences of up to 64 residues) and for a build beyond the thresholds the join
    serves (l_max = 9: text-chunk kernel), against oracle.lev_pairs edge by edge; the sweep down to 0."""
    rng = np.random.default_rng(64)
    strings = []
    for _ in range(300):
        n = int(rng.integers(20, 65))
        s = "".join("ACDEFGHIKLMNPQRSTVWY"[i] for i in rng.integers(0, 20, n))
        strings.append(s)
        for _ in range(3):
            t = list(s)
            for _ in range(int(rng.integers(1, 9))):
                q = int(rng.integers(0, len(t)))
                k = int(rng.integers(0, 3))
                if k == 0:
                    t[q] = "ACDEFGHIKLMNPQRSTVWY"[int(rng.integers(0, 20))]
                elif k == 1 and len(t) < 64:
                    t.insert(q, "W")
                elif len(t) > 1:
                    del t[q]
            strings.append("".join(t))
    res, ln = from_strings(strings)
    with pkg.TcrNet(0) as net:
        net.load(res, ln)
        for top in (9, 3):
            net.build(top)
            rp, cl, dg = net.copy_csr()
            rows = np.repeat(np.arange(len(strings), dtype=np.int64), np.diff(rp))
            want_d = oracle.lev_pairs(res, ln, np.stack([rows, cl.astype(np.int64)], axis=1)).astype(np.uint8)
            assert np.array_equal(net.edge_distances().cpu().numpy(), want_d) and want_d.max() == top
            for l in range(top - 1, -1, -2):
                assert net.restrict(l) == int((want_d <= l).sum())
                assert_same_network(net.copy_csr(), oracle.network(res, ln, l, tier=1)[:3])


def _query_network(oracle, d, n_query, l_max):
    """Oracle side of the rectangular mode: rows 0..n_query-1 against every other row."""
    pairs, _ = oracle.edges(d.residues, d.lengths, l_max, rows=np.arange(n_query), all_partners=True, tier=0)
    lo, hi = pairs.min(axis=1), pairs.max(axis=1)
    keys = np.unique((lo << 32) | hi)
    canon = np.stack([keys >> 32, keys & 0xffffffff], axis=1)
    return oracle.csr(canon, d.n)


@pytest.mark.parametrize("n_query", [1, 37, 700])
def test_query_mode(pkg, oracle, n_query):
    """NEXT-2 (antigen-specific networks): the first N_a rows are the queries;
    the build keeps exactly the edges with at least one query endpoint."""
    d = generate("cfg2", n=12000)
    # default: through the segment join (one pass over all rows, the emission keeps the pairs with a query row);
    # TCRNET_OPT_SEGMENT_JOIN = 0 / TCRNET_OPT_PREFIX_TRIE = 0 / l_max > 6: the two restricted passes of the trie /
    # text-chunk kernels
    for l_max, opts in ((0, {}), (1, {}), (2, {}), (3, {}), (4, {}), (5, {}), (6, {}), (7, {}),
                        (0, {pkg.OPT_SEGMENT_JOIN: 0}),
                        (1, {pkg.OPT_SEGMENT_JOIN: 0}), (2, {pkg.OPT_SEGMENT_JOIN: 0}), (3, {pkg.OPT_PREFIX_TRIE: 0}),
                        (4, {pkg.OPT_SEGMENT_JOIN: 0, pkg.OPT_TRIE_CHUNK: 512})):
        want = _query_network(oracle, d, n_query, l_max)
        with pkg.TcrNet(0) as net:
            for k, v in opts.items():
                net.set_option(k, v)
            net.set_option(pkg.OPT_N_QUERY, n_query)
            net.load(d.residues, d.lengths)
            net.build(l_max)
            got = net.copy_csr()
            st = net.get_stats()
            assert (st["join_mode"] >= 1) == (not opts and l_max <= 6)
            assert_same_network(got, want)
            assert (np.diff(got[0])[n_query:] == 0).all()                 # no row without a query endpoint
            assert st["pairs_all"] == n_query * (n_query - 1) // 2 + n_query * (d.n - n_query)
            # query mode off again on the same context -> the full network
            net.set_option(pkg.OPT_N_QUERY, 0)
            net.load(d.residues, d.lengths)
            net.build(l_max)
            full = net.copy_csr()
        assert int(full[0][-1]) >= int(want[0][-1])
        if l_max == 1:
            assert_same_network(full, oracle.network(d.residues, d.lengths, 1, tier=1)[:3])
