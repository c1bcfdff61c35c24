"""Writes tests/golden/<cfg>_l<l_max>_network.sha256: the WHOLE network of a BASELINE.json config, computed by the CPU
oracle alone, reduced to SHA-256 digests of the CSR + degree arrays.

    python tests/golden/make_config_hashes.py cfg3 cfg4 [--threads T] [--resume-dir DIR]

Imports only ``oracle`` and ``cdr3_synth`` (never the CUDA package): the stored values are the oracle's.
What is computed (section II.M: edge iff ``lev <= l_max``; section II.N: the
adjacency matrix, here its strict upper triangle as CSR; degrees): ``oracle.edges`` with
``tier=1`` over every row of the config, ``oracle.csr`` on the result.  Tier 1 is the full Wagner-Fischer table
plus the length filter and the paper's own row-minimum abort and is pinned equal to tier 0 in
tests/test_oracle_pins.py.  Cost on 8 cores: cfg3 (N = 200,000, l_max = 2) about 15-30 minutes, cfg4
(N = 800,000, l_max = 1) about an hour; cfg5 (N = 2,000,000, l_max = 3) would take about 125 core-hours and is
not stored (tests/test_parity_gpu.py checks it on sampled nodes and on every emitted edge instead).

The digests are over the little-endian bytes of ``row_ptr`` (int64[N+1]), ``col`` (int32[E]) and ``deg``
(int32[N]) - exactly what ``tcrnet_copy_csr`` hands back - and over their concatenation.  The rows are
processed in blocks so that a run can be interrupted and resumed (``--resume-dir`` keeps one ``.npy`` of pairs
per finished block; nothing is read from it unless it was written by this script for the same config).
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from cdr3_synth import CONFIGS, generate  # noqa: E402

BLOCK_ROWS = 10_000


def digest_lines(row_ptr: np.ndarray, col: np.ndarray, deg: np.ndarray) -> dict:
    rp = np.ascontiguousarray(row_ptr, dtype="<i8").tobytes()
    co = np.ascontiguousarray(col, dtype="<i4").tobytes()
    dg = np.ascontiguousarray(deg, dtype="<i4").tobytes()
    return {
        "sha256_row_ptr": hashlib.sha256(rp).hexdigest(),
        "sha256_col": hashlib.sha256(co).hexdigest(),
        "sha256_deg": hashlib.sha256(dg).hexdigest(),
        "sha256_all": hashlib.sha256(rp + co + dg).hexdigest(),
    }


def run(name: str, l_max: int, threads: int, resume_dir: str | None) -> str:
    cfg = CONFIGS[name]
    d = generate(name)
    n = d.n
    input_sha = hashlib.sha256(d.residues.tobytes() + d.lengths.astype("<i4").tobytes()).hexdigest()
    parts = []
    t_start = time.time()
    used = 0
    for b0 in range(0, n, BLOCK_ROWS):
        b1 = min(n, b0 + BLOCK_ROWS)
        path = None
        if resume_dir:
            os.makedirs(resume_dir, exist_ok=True)
            path = os.path.join(resume_dir, f"{name}_l{l_max}_{input_sha[:12]}_{b0}_{b1}.npy")
        if path and os.path.exists(path):
            pairs = np.load(path)
        else:
            pairs, used = oracle.edges(d.residues, d.lengths, l_max, rows=np.arange(b0, b1, dtype=np.int64),
                                       tier=1, threads=threads)
            if path:
                tmp = path + ".tmp.npy"
                np.save(tmp, pairs)
                os.replace(tmp, path)
        parts.append(pairs)
        print(f"{name}: rows {b0}..{b1} of {n}, {sum(p.shape[0] for p in parts)} edges, "
              f"{time.time() - t_start:.0f} s", flush=True)
    pairs = np.concatenate(parts) if parts else np.zeros((0, 2), dtype=np.int64)
    row_ptr, col, deg = oracle.csr(pairs, n)
    out = os.path.join(HERE, f"{name}_l{l_max}_network.sha256")
    lines = {
        "config": name, "n": n, "l_max": l_max, "seed": cfg.seed, "sha256_input": input_sha,
        "n_edges": int(row_ptr[-1]), "max_degree": int(deg.max()), "sum_degree": int(deg.sum(dtype=np.int64)),
        "n_isolated": int((deg == 0).sum()),
    }
    lines.update(digest_lines(row_ptr, col, deg))
    with open(out, "w") as f:
        f.write(f"# whole-network digests of BASELINE.json {name}, l_max = {l_max}; written by\n"
                f"# tests/golden/make_config_hashes.py from the tier-1 CPU oracle alone (PAPER.md:297, 301-318, 224)\n")
        for k, v in lines.items():
            f.write(f"{k} {v}\n")
    print(f"{name}: wrote {out} ({lines['n_edges']} edges, {time.time() - t_start:.0f} s, threads {used})", flush=True)
    return out


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("configs", nargs="+", choices=sorted(CONFIGS))
    ap.add_argument("--l-max", type=int, default=None, help="default: the config's (first) threshold")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--resume-dir", default=None)
    a = ap.parse_args()
    for name in a.configs:
        run(name, CONFIGS[name].l_max[0] if a.l_max is None else a.l_max, a.threads, a.resume_dir)


if __name__ == "__main__":
    main()
