"""Pins for the CPU oracle (oracle/): none of these re-use the oracle's formula.

Each test names the part of oracle/tcrnet_oracle.c it pins and the mistake it
would catch.  All CPU, seconds.
"""
import itertools
import os
from collections import deque

import numpy as np
import pytest

import oracle
from cdr3_synth import generate
from cdr3_synth.generator import from_strings

RNG = np.random.default_rng(7)
AA = "ACDEFGHIKLMNPQRSTVWY"


def rand_str(n, alphabet=AA):
    return "".join(alphabet[i] for i in RNG.integers(0, len(alphabet), n))


# ------------------------------------------------------------------ lev: printed values
def test_golden_examples(golden_dir):
    """PAPER.md:293 ACCA/ACGG = 2, kitten/sitting = 3, base cases (tests/golden/lev_examples.txt)."""
    n = 0
    for line in open(os.path.join(golden_dir, "lev_examples.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        a, b, d = line.split()
        a = "" if a == "-" else a
        b = "" if b == "-" else b
        assert oracle.lev(a, b) == int(d), (a, b)
        assert oracle.lev(b, a) == int(d), (b, a)
        n += 1
    assert n == 6


# ------------------------------------------------------------------ lev: exhaustive search
def _bfs_distances(universe, alphabet, max_len):
    """Edit distance by breadth-first search over single-character edits.

    Definition-level: the minimum number of insertions, deletions and
    substitutions.  Restricting intermediate strings to length <= max_len and
    to the alphabet loses nothing (do deletions before insertions; foreign
    letters never help)."""
    def neighbours(s):
        out = set()
        for i in range(len(s)):
            out.add(s[:i] + s[i + 1:])
            for c in alphabet:
                out.add(s[:i] + c + s[i + 1:])
        if len(s) < max_len:
            for i in range(len(s) + 1):
                for c in alphabet:
                    out.add(s[:i] + c + s[i:])
        out.discard(s)
        return out

    nb = {s: neighbours(s) for s in universe}
    dist = {}
    for src in universe:
        d = {src: 0}
        q = deque([src])
        while q:
            s = q.popleft()
            for t in nb[s]:
                if t not in d:
                    d[t] = d[s] + 1
                    q.append(t)
        dist[src] = d
    return dist


@pytest.mark.parametrize("alphabet,max_len", [("AB", 5), ("ABC", 4)])
def test_exhaustive_edit_script_search(alphabet, max_len):
    """All pairs of strings of length <= 5 (binary) / <= 4 (ternary): table == BFS over edit scripts.
    Catches a dropped term, a wrong index or base case anywhere in the recurrence."""
    universe = [""] + ["".join(p) for k in range(1, max_len + 1) for p in itertools.product(alphabet, repeat=k)]
    dist = _bfs_distances(universe, alphabet, max_len)
    for a in universe:
        for b in universe:
            assert oracle.lev(a, b) == dist[a][b], (a, b)


# ------------------------------------------------------------------ lev: axioms, closed forms, invariances
def test_identity_empty_symmetry_bounds():
    for _ in range(300):
        m, n = RNG.integers(0, 40, 2)
        a, b = rand_str(m), rand_str(n)
        d = oracle.lev(a, b)
        assert oracle.lev(a, a) == 0
        assert oracle.lev(a, "") == m and oracle.lev("", a) == m
        assert d == oracle.lev(b, a)
        assert abs(m - n) <= d <= max(m, n)
        if m == n:
            assert d <= sum(x != y for x, y in zip(a, b))  # lev <= Hamming (reading Q6)
        if a != b:
            assert d >= 1


def test_triangle_inequality_random_triples():
    for _ in range(400):
        # small alphabet + short strings make the inequality tight often
        a, b, c = (rand_str(RNG.integers(0, 12), "ACD") for _ in range(3))
        assert oracle.lev(a, c) <= oracle.lev(a, b) + oracle.lev(b, c)


def test_closed_forms():
    for m in range(0, 30, 3):
        for n in range(0, 30, 4):
            assert oracle.lev("A" * m, "A" * n) == abs(m - n)
            assert oracle.lev("A" * m, "C" * n) == max(m, n)
    # disjoint alphabets: nothing can match
    assert oracle.lev("ACDEF", "GHIKLMN") == 7
    # one string a subsequence of the other: distance = length difference
    s = "CASSLGQGNTEAFF"
    sub = "".join(ch for k, ch in enumerate(s) if k not in (3, 7, 8))
    assert oracle.lev(s, sub) == 3 and oracle.lev(sub, s) == 3


def test_invariances():
    perm = dict(zip(AA, RNG.permutation(list(AA))))
    for _ in range(200):
        a, b = rand_str(RNG.integers(1, 25)), rand_str(RNG.integers(1, 25))
        d = oracle.lev(a, b)
        assert oracle.lev(a[::-1], b[::-1]) == d  # reversal (catches transposed / shifted indexing)
        assert oracle.lev("".join(perm[c] for c in a), "".join(perm[c] for c in b)) == d
        p, s = rand_str(RNG.integers(0, 6)), rand_str(RNG.integers(0, 6))
        assert oracle.lev(p + a + s, p + b + s) == d  # common affixes cancel


def test_exact_distance_by_bag_bound():
    """k edits with letters foreign to the string: upper bound k (the script) meets the
    bag-distance lower bound k, so the distance is exactly k without any DP."""
    for _ in range(200):
        n = int(RNG.integers(6, 30))
        a = list(rand_str(n, "ACDEFGHIKL"))
        k = int(RNG.integers(0, 6))
        b = a[:]
        pos = sorted(RNG.choice(n, size=k, replace=False), reverse=True)
        kinds = RNG.integers(0, 2, k)
        for p, kind in zip(pos, kinds):
            foreign = "WY"[int(RNG.integers(0, 2))]
            if kind == 0:
                b[p] = foreign  # substitution
            else:
                b.insert(p, foreign)  # insertion
        assert oracle.lev("".join(a), "".join(b)) == k
        assert oracle.lev("".join(b), "".join(a)) == k


# ------------------------------------------------------------------ threshold, duplicates, edges
def test_threshold_is_less_or_equal():
    """PAPER.md:297 'l <= l_max' (reading Q2, not Listing 1's '<'): a pair at distance exactly
    l_max is an edge, at l_max + 1 it is not."""
    base = "CASSLGQGNTEAFF"
    for k in range(0, 5):
        other = "".join("W" if i < k else ch for i, ch in enumerate(base))  # exactly k substitutions
        res, ln = from_strings([base, other])
        for l_max in range(0, 6):
            pairs, _ = oracle.edges(res, ln, l_max)
            assert (pairs.shape[0] == 1) == (k <= l_max), (k, l_max)


def test_duplicates_form_complete_graph():
    """Reading Q3: one node per row; r copies give K_r for every l_max >= 0 (d = 0 <= l_max)."""
    r = 7
    res, ln = from_strings(["CASSF"] * r + ["CWWWWWWWF"])
    for l_max in (0, 1, 3):
        pairs, _ = oracle.edges(res, ln, l_max)
        want = [(i, j) for i in range(r) for j in range(i + 1, r)]
        assert [tuple(p) for p in pairs] == want
        row_ptr, col, deg = oracle.csr(pairs, r + 1)
        assert deg.tolist() == [r - 1] * r + [0]


def test_lmax_zero_equals_exact_match_join():
    d = generate("cfg1")
    pairs, _ = oracle.edges(d.residues, d.lengths, 0)
    groups = {}
    for i, s in enumerate(d.strings()):
        groups.setdefault(s, []).append(i)
    want = sorted((a, b) for g in groups.values() for a, b in itertools.combinations(g, 2))
    assert [tuple(p) for p in pairs] == want
    assert len(want) > 100  # the workload really has duplicates


def test_paper_five_node_example(golden_dir):
    """edge list -> adjacency matrix (Eq. 17) -> CSR / degrees."""
    fields = {}
    matrix = []
    mode = None
    for line in open(os.path.join(golden_dir, "paper_adjacency_example.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.endswith(":") and line[:-1] == "matrix":
            mode = "matrix"
            continue
        if ":" in line:
            k, v = line.split(":")
            fields[k] = [int(x) for x in v.split()]
            mode = None
        elif mode == "matrix":
            matrix.append([int(x) for x in line.split()])
    A = np.array(matrix)
    e1 = np.array(fields["edges_1based"]).reshape(-1, 2)
    row_ptr, col, deg = oracle.csr(e1 - 1, 5)
    assert row_ptr.tolist() == fields["row_ptr"]
    assert col.tolist() == fields["col"]
    assert deg.tolist() == fields["deg"]
    # CSR -> symmetric matrix equals the printed matrix; degrees are its row sums
    B = np.zeros((5, 5), dtype=int)
    for u in range(5):
        for k in range(row_ptr[u], row_ptr[u + 1]):
            B[u, col[k]] = B[col[k], u] = 1
    assert (A == B).all() and (A.sum(1) == deg).all() and (np.diag(A) == 0).all()
    # the same graph realised by strings at l_max = 1 goes through the whole oracle path
    res, ln = from_strings(["AAAA", "AAAB", "AACA", "AEDB", "AADB"])
    rp, cl, dg, _ = oracle.network(res, ln, 1)
    assert rp.tolist() == fields["row_ptr"] and cl.tolist() == fields["col"] and dg.tolist() == fields["deg"]


def test_csr_rejects_unsorted_or_lower_triangle():
    with pytest.raises(ValueError):
        oracle.csr(np.array([[1, 2], [0, 3]]), 4)
    with pytest.raises(ValueError):
        oracle.csr(np.array([[2, 1]]), 4)
    with pytest.raises(ValueError):
        oracle.csr(np.array([[0, 1], [0, 1]]), 4)


def test_csr_invariants_and_dense_rebuild():
    d = generate("cfg1", n=300)
    for l_max in (0, 1, 2, 4):
        row_ptr, col, deg, _ = oracle.network(d.residues, d.lengths, l_max)
        E = int(row_ptr[-1])
        assert row_ptr[0] == 0 and (np.diff(row_ptr) >= 0).all() and col.size == E
        assert deg.sum() == 2 * E
        A = np.zeros((d.n, d.n), dtype=np.int8)
        for u in range(d.n):
            c = col[row_ptr[u]:row_ptr[u + 1]]
            assert (c > u).all() and (np.diff(c) > 0).all()
            A[u, c] = 1
        A = A + A.T
        assert (A.sum(1) == deg).all()
        # brute force over the full matrix with single calls
        s = d.strings()
        for u in RNG.integers(0, d.n, 12):
            for v in range(d.n):
                if u != v:
                    assert A[u, v] == (oracle.lev(s[u], s[v]) <= l_max)


def test_monotone_in_lmax_and_generator_lower_bound():
    d = generate("cfg1")
    prev = set()
    for l_max in (0, 1, 2, 3):
        pairs, _ = oracle.edges(d.residues, d.lengths, l_max)
        cur = set(map(tuple, pairs))
        assert prev <= cur  # E(l) subset of E(l+1)
        prev = cur
        # generator-linked lower bound: same family, edits sum <= l_max  =>  edge
        fam = {}
        for i in range(d.n):
            if d.family[i] >= 0:
                fam.setdefault(int(d.family[i]), []).append(i)
        must = 0
        for rows in fam.values():
            for a, b in itertools.combinations(rows, 2):
                if d.n_edits[a] + d.n_edits[b] <= l_max:
                    assert (a, b) in cur
                    must += 1
        assert must > 0


def _within_one(a: bytes, b: bytes) -> bool:
    """Textbook l_max = 1 test: equal length -> Hamming <= 1; lengths differ by one -> the
    shorter is the longer with one character deleted; otherwise no."""
    if len(a) == len(b):
        return sum(x != y for x, y in zip(a, b)) <= 1
    if abs(len(a) - len(b)) != 1:
        return False
    if len(a) < len(b):
        a, b = b, a
    k = 0
    while k < len(b) and a[k] == b[k]:
        k += 1
    return a[k + 1:] == b[k:]


def test_lmax1_textbook_characterisation_cfg1():
    """The whole edge set of config 1 at l_max = 1 against an independent 15-line checker."""
    d = generate("cfg1")
    s = d.strings()
    want = [(i, j) for i in range(d.n) for j in range(i + 1, d.n)
            if abs(len(s[i]) - len(s[j])) <= 1 and _within_one(s[i], s[j])]
    pairs, _ = oracle.edges(d.residues, d.lengths, 1)
    assert [tuple(p) for p in pairs] == want
    assert 2000 < len(want) < 20000


# ------------------------------------------------------------------ tier 1, sampled-row mode
def test_tier1_equals_tier0():
    d = generate("cfg1")
    for l_max in (0, 1, 2, 3, 6):
        p0, _ = oracle.edges(d.residues, d.lengths, l_max, tier=0)
        p1, _ = oracle.edges(d.residues, d.lengths, l_max, tier=1)
        assert np.array_equal(p0, p1)
    d = generate("cfg2", n=6000)
    rows = np.sort(RNG.choice(d.n, 150, replace=False))
    for l_max in (1, 2):
        p0, _ = oracle.edges(d.residues, d.lengths, l_max, rows=rows, all_partners=True, tier=0)
        p1, _ = oracle.edges(d.residues, d.lengths, l_max, rows=rows, all_partners=True, tier=1)
        assert np.array_equal(p0, p1) and p0.shape[0] > 0


def test_abort_variant_matches_when_within_threshold():
    for _ in range(500):
        a, b = rand_str(RNG.integers(0, 20), "ACD"), rand_str(RNG.integers(0, 20), "ACD")
        d = oracle.lev(a, b)
        for l_max in (0, 1, 2, 5):
            da = oracle.lev_abort(a, b, l_max)
            assert (da <= l_max) == (d <= l_max)
            if d <= l_max:
                assert da == d


def test_rows_and_all_partners_modes():
    d = generate("cfg1", n=400)
    full, _ = oracle.edges(d.residues, d.lengths, 2)
    rows = np.array([3, 77, 200, 399])
    part, _ = oracle.edges(d.residues, d.lengths, 2, rows=rows)
    assert np.array_equal(part, full[np.isin(full[:, 0], rows)])
    nb, _ = oracle.edges(d.residues, d.lengths, 2, rows=rows, all_partners=True)
    for r in rows:
        want = sorted(set(full[full[:, 0] == r, 1]) | set(full[full[:, 1] == r, 0]))
        assert nb[nb[:, 0] == r, 1].tolist() == want


def test_thread_count_does_not_change_result():
    d = generate("cfg1", n=500)
    p1, t1 = oracle.edges(d.residues, d.lengths, 1, threads=1)
    p3, t3 = oracle.edges(d.residues, d.lengths, 1, threads=3)
    assert t1 == 1 and t3 == 3 and np.array_equal(p1, p3)


def test_lev_pairs_is_the_same_table_pair_by_pair():
    """oracle.lev_pairs (the batched driver the large-config parity tests use) against the breadth-first search over
    edit scripts (all pairs of binary strings of length <= 4, laid out as rows) and against construction: a string
    and the same string after k substitutions at distinct positions of a disjoint alphabet has distance exactly k."""
    universe = [""] + ["".join(p) for k in range(1, 5) for p in itertools.product("AB", repeat=k)]
    dist = _bfs_distances(universe, "AB", 4)
    rows = [s for s in universe if s]
    res, ln = from_strings(rows)
    pairs = np.array([(i, j) for i in range(len(rows)) for j in range(len(rows))], dtype=np.int64)
    got = oracle.lev_pairs(res, ln, pairs, threads=2)
    want = np.array([dist[rows[i]][rows[j]] for i, j in pairs], dtype=np.int32)
    assert np.array_equal(got, want)
    base = [rand_str(int(RNG.integers(6, 30)), "ACDEF") for _ in range(200)]
    ks = [int(RNG.integers(0, len(s) + 1)) for s in base]
    changed = []
    for s, k in zip(base, ks):
        t = list(s)
        for q in RNG.choice(len(s), k, replace=False):
            t[q] = "W"
        changed.append("".join(t))
    res, ln = from_strings(base + changed)
    pairs = np.array([(i, i + len(base)) for i in range(len(base))], dtype=np.int64)
    assert oracle.lev_pairs(res, ln, pairs).tolist() == ks
    with pytest.raises(ValueError):
        oracle.lev_pairs(res, ln, np.array([[0, 2 * len(base)]], dtype=np.int64))


@pytest.mark.skipif(os.environ.get("TCRNET_ORACLE_SANITIZE") == "1", reason="already inside the sanitizer run")
def test_pins_under_address_and_ub_sanitizers():
    """the oracle under -fsanitize=address,undefined.  A subprocess builds
    oracle/libtcrnet_oracle_asan.so and runs the quick pins (tables, edge lists, CSR, threads) against it; any
    out-of-bounds access, use after free, signed overflow or misaligned access in the C sources aborts it."""
    import subprocess
    import sys
    from oracle import build as ob
    runtime = ob.sanitizer_runtime()
    if not os.path.isabs(runtime) or not os.path.exists(runtime):
        pytest.skip("gcc has no libasan.so here")
    env = dict(os.environ)
    env.update({ob.SANITIZE_ENV: "1", "LD_PRELOAD": runtime, "ASAN_OPTIONS": "detect_leaks=0",
                "UBSAN_OPTIONS": "halt_on_error=1:print_stacktrace=1", "OMP_NUM_THREADS": "4"})
    sel = ("golden_examples or identity_empty or closed_forms or threshold_is_less or duplicates_form or "
           "lmax_zero or five_node or csr_rejects or csr_invariants or rows_and_all_partners or thread_count or "
           "lev_pairs or abort_variant")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                        os.path.join(root, "tests", "test_oracle_pins.py"),
                        os.path.join(root, "tests", "test_observables_pins.py"), "-k", sel + " or observables or closed or paper"],
                       cwd=root, env=env, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "passed" in r.stdout
