"""Family-structured random CDR3-beta-like sequences, fully vectorised and seeded.

Recipe (BASELINE.json `configs`; restated in DESIGN.md):

1. ``rng = numpy.random.Generator(numpy.random.PCG64(seed))``; every draw below
   comes from it, in the order written here.
2. ``n_dup = round(dup * N)`` rows will be copies; ``n_base = N - n_dup``.
3. Seeds: ``n_seeds`` sequences.  Length ``clip(rint(Normal(mu, sigma)), lo,
   hi)``.  First residue 'C', last residue 'F' (the stress input ``cfg4_cass``:
   first residues 'CASS', last 'EQYF'), the rest i.i.d. from the
   residue law of that seed (uniform over the 20 standard amino acids of
   PAPER.md:211, or — config 5 — with probability ``zipf_frac`` a Zipf(s=1.1)
   law over the same 20 letters in ``AA20`` order).
4. Seed ``s`` spawns ``Poisson(lam) + 1`` variants (families are laid out
   seed by seed and cut at ``n_base`` rows).  A variant is the seed with
   ``Poisson(1)`` random edits; an edit is a substitution, an insertion or a
   deletion (equiprobable) at a uniform position with a residue from the seed's
   law; an edit that would leave ``[lo, hi]`` is skipped (and not counted).
5. If the families give fewer than ``n_base`` rows, the rest are independent
   random sequences from the same length / residue law (family id -1).
6. ``n_dup`` copies of uniformly chosen base rows are appended.
7. One uniform random permutation of the N rows is applied.

Output is the caller-facing form of the boundary: concatenated ASCII residues,
``int32`` lengths, plus bookkeeping (family id, number of applied edits) that
tests use for the generator-linked lower bound (two rows of one family whose
edit counts sum to <= l_max must be joined by an edge).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Tuple

import numpy as np

AA20 = b"ACDEFGHIKLMNPQRSTVWY"  # the alphabet of PAPER.md:211
_AA = np.frombuffer(AA20, dtype=np.uint8)
_SEED_BASE = 20211214  # arXiv submission date of the paper; + config index


@dataclass(frozen=True)
class SynthConfig:
    name: str
    index: int  # 1-based index into BASELINE.json `configs`
    n: int
    l_max: Tuple[int, ...]
    n_seeds: int
    lam: float
    mu: float
    sigma: float
    lo: int
    hi: int
    dup: float
    zipf_frac: float = 0.0
    prefix: bytes = b"C"   # conserved first residues of every seed / independent sequence
    suffix: bytes = b"F"   # conserved last residues

    @property
    def seed(self) -> int:
        return _SEED_BASE + self.index


CONFIGS: Dict[str, SynthConfig] = {
    c.name: c
    for c in (
        SynthConfig("cfg1", 1, 2_000, (1,), 200, 9.0, 15.0, 2.0, 8, 25, 0.05),
        SynthConfig("cfg2", 2, 50_000, (1, 2), 2_000, 24.0, 15.0, 2.0, 8, 25, 0.05),
        SynthConfig("cfg3", 3, 200_000, (2,), 8_000, 24.0, 15.0, 2.5, 6, 30, 0.05),
        SynthConfig("cfg4", 4, 800_000, (1,), 30_000, 24.0, 15.0, 2.0, 8, 25, 0.03),
        SynthConfig("cfg5", 5, 2_000_000, (3,), 60_000, 24.0, 16.0, 3.0, 5, 40, 0.05, 0.10),
        # Stress input, NOT a BASELINE.json config: config 4 with the conserved ends real CDR3-beta rows have (V gene:
        # "CASS...", J gene: "...EQYF"), so that prefixes / suffixes carry no information (bench.py `detail`, DESIGN.md
        # section 6).  lo >= len(prefix) + len(suffix).
        SynthConfig("cfg4_cass", 14, 800_000, (1,), 30_000, 24.0, 15.0, 2.0, 8, 25, 0.03, 0.0, b"CASS", b"EQYF"),
    )
}


def get_config(name: str) -> SynthConfig:
    return CONFIGS[name]


@dataclass
class SynthData:
    config: SynthConfig
    residues: np.ndarray  # uint8[sum(lengths)], ASCII, concatenated row by row
    lengths: np.ndarray  # int32[N]
    offsets: np.ndarray  # int64[N+1], exclusive prefix sum of lengths
    family: np.ndarray  # int32[N], seed index or -1
    n_edits: np.ndarray  # int32[N], edits actually applied to the seed
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.lengths.shape[0])

    def row(self, i: int) -> bytes:
        return self.residues[self.offsets[i] : self.offsets[i + 1]].tobytes()

    def strings(self):
        return [self.row(i) for i in range(self.n)]


def _lengths(rng, k, cfg):
    return np.clip(np.rint(rng.normal(cfg.mu, cfg.sigma, k)), cfg.lo, cfg.hi).astype(np.int64)


def _residue_cdf(zipf: bool) -> np.ndarray:
    if zipf:
        p = 1.0 / np.arange(1, 21, dtype=np.float64) ** 1.1
    else:
        p = np.ones(20, dtype=np.float64)
    c = np.cumsum(p / p.sum())
    c[-1] = 1.0
    return c


_CDF = (_residue_cdf(False), _residue_cdf(True))


def _draw_residues(rng, is_zipf: np.ndarray, shape) -> np.ndarray:
    """i.i.d. residues, one law per leading row (is_zipf is bool[rows])."""
    u = rng.random(shape)
    idx_u = np.minimum(np.searchsorted(_CDF[0], u, side="right"), 19)
    if is_zipf.any():
        idx_z = np.minimum(np.searchsorted(_CDF[1], u, side="right"), 19)
        sel = is_zipf.reshape((-1,) + (1,) * (u.ndim - 1))
        idx_u = np.where(sel, idx_z, idx_u)
    return _AA[idx_u]


def _random_sequences(rng, k, cfg):
    """k independent sequences: (matrix uint8[k, hi], lengths, is_zipf)."""
    ln = _lengths(rng, k, cfg)
    zipf = rng.random(k) < cfg.zipf_frac if cfg.zipf_frac > 0 else np.zeros(k, dtype=bool)
    mat = _draw_residues(rng, zipf, (k, cfg.hi))
    for q, ch in enumerate(cfg.prefix):
        mat[:, q] = ch
    for q, ch in enumerate(reversed(cfg.suffix)):
        mat[np.arange(k), ln - 1 - q] = ch
    col = np.arange(cfg.hi)[None, :]
    mat[col >= ln[:, None]] = 0
    return mat, ln, zipf


def _apply_edit_round(rng, mat, ln, zipf, rows, cfg):
    """One edit on each of `rows` (in place).  Returns bool[rows]: applied."""
    k = rows.shape[0]
    kind = rng.integers(0, 3, k)  # 0 substitution, 1 insertion, 2 deletion
    u = rng.random(k)
    res = _draw_residues(rng, zipf[rows], (k,))
    cur = ln[rows]
    applied = np.ones(k, dtype=bool)
    applied[(kind == 1) & (cur >= cfg.hi)] = False
    applied[(kind == 2) & (cur <= cfg.lo)] = False
    span = np.where(kind == 1, cur + 1, cur)  # insertion has len+1 slots
    pos = np.minimum((u * span).astype(np.int64), span - 1)
    col = np.arange(cfg.hi)[None, :]

    m = applied & (kind == 0)
    if m.any():
        mat[rows[m], pos[m]] = res[m]
    m = applied & (kind == 1)
    if m.any():
        r, p = rows[m], pos[m][:, None]
        old = mat[r]
        shifted = np.concatenate([old[:, :1], old[:, :-1]], axis=1)  # old[c-1]
        new = np.where(col < p, old, np.where(col == p, res[m][:, None], shifted))
        mat[r] = new
        ln[r] += 1
    m = applied & (kind == 2)
    if m.any():
        r, p = rows[m], pos[m][:, None]
        old = mat[r]
        shifted = np.concatenate([old[:, 1:], np.zeros_like(old[:, :1])], axis=1)  # old[c+1]
        mat[r] = np.where(col < p, old, shifted)
        ln[r] -= 1
    return applied


def generate(cfg: SynthConfig | str, n: int | None = None, seed: int | None = None) -> SynthData:
    """Generate the workload of `cfg` (optionally overriding N and the seed)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    if n is not None and n != cfg.n:
        scale = n / cfg.n
        cfg = SynthConfig(cfg.name, cfg.index, n, cfg.l_max, max(1, int(round(cfg.n_seeds * scale))),
                          cfg.lam, cfg.mu, cfg.sigma, cfg.lo, cfg.hi, cfg.dup, cfg.zipf_frac, cfg.prefix, cfg.suffix)
    rng = np.random.Generator(np.random.PCG64(cfg.seed if seed is None else seed))
    N = cfg.n
    n_dup = int(round(cfg.dup * N))
    n_base = N - n_dup

    seed_mat, seed_len, seed_zipf = _random_sequences(rng, cfg.n_seeds, cfg)
    counts = rng.poisson(cfg.lam, cfg.n_seeds) + 1
    fam = np.repeat(np.arange(cfg.n_seeds), counts)[:n_base]
    n_fam = fam.shape[0]

    mat = np.zeros((n_base, cfg.hi), dtype=np.uint8)
    ln = np.zeros(n_base, dtype=np.int64)
    zipf = np.zeros(n_base, dtype=bool)
    family = np.full(n_base, -1, dtype=np.int32)
    n_edits = np.zeros(n_base, dtype=np.int32)
    mat[:n_fam] = seed_mat[fam]
    ln[:n_fam] = seed_len[fam]
    zipf[:n_fam] = seed_zipf[fam]
    family[:n_fam] = fam

    want = rng.poisson(1.0, n_fam)
    r = 0
    while True:
        rows = np.nonzero(want > r)[0]
        if rows.size == 0:
            break
        applied = _apply_edit_round(rng, mat, ln, zipf, rows, cfg)
        n_edits[rows[applied]] += 1
        r += 1

    if n_fam < n_base:
        fm, fl, fz = _random_sequences(rng, n_base - n_fam, cfg)
        mat[n_fam:], ln[n_fam:], zipf[n_fam:] = fm, fl, fz

    if n_dup:
        src = rng.integers(0, n_base, n_dup)
        mat = np.concatenate([mat, mat[src]])
        ln = np.concatenate([ln, ln[src]])
        family = np.concatenate([family, family[src]])
        n_edits = np.concatenate([n_edits, n_edits[src]])

    perm = rng.permutation(N)
    mat, ln, family, n_edits = mat[perm], ln[perm], family[perm], n_edits[perm]

    col = np.arange(cfg.hi)[None, :]
    residues = np.ascontiguousarray(mat[col < ln[:, None]])
    offsets = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(ln, out=offsets[1:])
    return SynthData(cfg, residues, ln.astype(np.int32), offsets, family, n_edits,
                     meta={"n_family_rows": int(n_fam), "n_dup": n_dup, "seed": cfg.seed if seed is None else seed})


def from_strings(strings) -> Tuple[np.ndarray, np.ndarray]:
    """Boundary form (residues, lengths) of a list of bytes/str — test helper."""
    bs = [s.encode() if isinstance(s, str) else bytes(s) for s in strings]
    lengths = np.array([len(b) for b in bs], dtype=np.int32)
    residues = np.frombuffer(b"".join(bs), dtype=np.uint8).copy()
    return residues, lengths
