"""The seeded input generator (cdr3_synth/): determinism and the shapes BASELINE.json states."""
import hashlib

import numpy as np

from cdr3_synth import AA20, CONFIGS, generate


def test_deterministic_and_shaped():
    a, b = generate("cfg1"), generate("cfg1")
    assert np.array_equal(a.residues, b.residues) and np.array_equal(a.lengths, b.lengths)
    assert a.n == 2000 and a.offsets[-1] == a.residues.size
    assert a.lengths.min() >= 8 and a.lengths.max() <= 25
    assert set(np.unique(a.residues)) <= set(AA20)
    assert abs(a.lengths.mean() - 15.0) < 0.3
    assert a.meta["n_dup"] == 100
    # every family row is within n_edits edits of its seed, so rows start with C / end with F mostly
    s = a.strings()
    assert sum(x[:1] == b"C" for x in s) > 0.9 * a.n and sum(x[-1:] == b"F" for x in s) > 0.9 * a.n
    assert len(set(s)) < a.n  # duplicates exist (reading Q3 is exercised)


def test_other_seed_differs_and_scaling_override():
    a, b = generate("cfg1"), generate("cfg1", seed=1)
    assert not np.array_equal(a.residues[:100], b.residues[:100])
    c = generate("cfg4", n=5000)
    assert c.n == 5000 and c.lengths.min() >= 8 and c.lengths.max() <= 25


def test_config_table_matches_baseline_json():
    want = {"cfg1": (2_000, (1,), 8, 25), "cfg2": (50_000, (1, 2), 8, 25), "cfg3": (200_000, (2,), 6, 30),
            "cfg4": (800_000, (1,), 8, 25), "cfg5": (2_000_000, (3,), 5, 40)}
    for k, (n, lm, lo, hi) in want.items():
        c = CONFIGS[k]
        assert (c.n, c.l_max, c.lo, c.hi) == (n, lm, lo, hi)
    assert CONFIGS["cfg5"].zipf_frac == 0.10 and CONFIGS["cfg4"].dup == 0.03


def test_cfg5_shape_small():
    d = generate("cfg5", n=20000)
    assert d.lengths.min() >= 5 and d.lengths.max() <= 40
    # Zipf rows skew the composition towards the first letters of AA20
    counts = np.bincount(d.residues, minlength=128)[list(AA20)]
    assert counts[0] > counts[10]


def test_stream_is_pinned():
    """A change to the generator changes every expected value downstream: pin its output."""
    d = generate("cfg1")
    h = hashlib.sha256(d.residues.tobytes() + d.lengths.tobytes()).hexdigest()
    assert h == open(__file__.replace("test_synth.py", "golden/cfg1_input.sha256")).read().split()[0]


def test_stored_network_digests_belong_to_the_generated_inputs():
    """tests/golden/<cfg>_l<l_max>_network.sha256 (written by tests/golden/make_config_hashes.py from the oracle alone)
    exist for config 1, 3 and 4 and were computed on exactly the rows the generator produces today."""
    import hashlib
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    for name, l_max in (("cfg1", 1), ("cfg3", 2), ("cfg4", 1)):
        path = os.path.join(here, f"{name}_l{l_max}_network.sha256")
        assert os.path.exists(path), path
        kv = dict(line.split() for line in open(path) if line.strip() and not line.startswith("#"))
        d = generate(name)
        assert int(kv["n"]) == d.n and int(kv["l_max"]) == l_max
        assert kv["sha256_input"] == hashlib.sha256(d.residues.tobytes() + d.lengths.astype("<i4").tobytes()).hexdigest()
        assert int(kv["sum_degree"]) == 2 * int(kv["n_edges"])
        for k in ("sha256_row_ptr", "sha256_col", "sha256_deg", "sha256_all"):
            assert len(kv[k]) == 64
