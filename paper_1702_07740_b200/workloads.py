"""Seeded synthetic workloads: the five BASELINE.json configs (codes + frames).

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench.py, smoke).  It holds none of
the decoder's arithmetic: it draws base matrices, random words, their syndromes and BIAWGN channel LLRs with
numpy only.  It imports neither `oracle/` nor the CUDA binding.

Conventions (citations are /root/reference/PAPER.md lines, "P:NNN"):

* Base matrix `base_shifts[mb][nb]`, int32: -1 = all-zero ZxZ block, p in [0,Z) = the ZxZ identity with every row
  cyclically shifted right by p (paper entry i = p+1): check R*Z + r is connected to variable
  C*Z + ((r + p) mod Z).  Rows are checks, columns are variables.
* Structure (Fig. 11; BASELINE.json configs): `n_core` dense "core" columns on the left, then a long
  unshifted diagonal of degree-1 variables: column j >= n_core connects only to row j - n_core + top_rows, shift 0.
  Each core column has `top_deg` edges to distinct random rows among the `top_rows` top rows and `low_deg` edges to
  the lower rows, dealt so that every lower row receives exactly 2 core edges (readings S11, S14).
* Frames: x uniform bits, s = H x mod 2, y = (1 - 2x) + N(0, sigma^2), LLR = 2 y / sigma^2 in fp32 (P:344 with one
  sigma per frame).  sigma comes from `SIGMA_STAR` (BIAWGN capacity threshold, written by
  `oracle/make_sigma_table.py`, which calls only `oracle/`) and the config's gap in dB.

These inputs stand in for the paper's unpublished parity-check matrices and QKD data.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, Tuple

import numpy as np

CODE_SEED_BASE = 17020774000  # + config index
FRAME_SEED_BASE = 17020775000  # + 1000 * config index + frame index (+ 100 * snr point for config 5)

# sigma* with C_BIAWGN(sigma*) = R, i.e. the channel noise std-dev at capacity for rate R.
# Written by oracle/make_sigma_table.py (numerical integration in oracle/capacity.py); tests/test_capacity.py
# re-derives them and compares.  Keys are code rates.
SIGMA_STAR: Dict[float, float] = {
    0.1: 2.5927695318,
    0.05: 3.7325617743,
    0.02: 5.9640225450,
}


@dataclass(frozen=True)
class CodeSpec:
    """Shape of one BASELINE.json code family."""
    name: str
    nb: int          # base columns
    mb: int          # base rows
    Z: int           # lifting size
    n_core: int      # core (degree > 1) columns
    top_rows: int    # rows holding the `top_deg` edges of each core column
    top_deg: int
    low_deg: int     # edges of each core column into the lower rows
    rate: float      # design rate 1 - mb/nb
    seed: int

    @property
    def n(self) -> int:
        return self.nb * self.Z

    @property
    def m(self) -> int:
        return self.mb * self.Z


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: a code, a channel point and the decode arguments."""
    index: int
    code: CodeSpec
    n_frames: int
    max_iter: int
    early_stop: int
    gaps_db: Tuple[float, ...]      # dB above BIAWGN capacity, one entry per SNR point
    description: str = ""


def _spec(name, nb, mb, Z, n_core, top_rows, top_deg, low_deg, rate, idx) -> CodeSpec:
    return CodeSpec(name, nb, mb, Z, n_core, top_rows, top_deg, low_deg, rate, CODE_SEED_BASE + idx)


CONFIGS: Dict[int, Config] = {
    1: Config(1, _spec("r0.10_80x72_Z32", 80, 72, 32, 16, 8, 3, 8, 0.1, 1), 16, 50, 0, (1.5,),
              "tiny rate-0.1 code, 16 frames, 50 flooding iterations, early stop off"),
    2: Config(2, _spec("r0.10_80x72_Z12500", 80, 72, 12500, 16, 8, 3, 8, 0.1, 2), 1, 200, 1, (0.5,),
              "rate-0.1 n=1e6, 1 frame, max 200 iterations, early stop on"),
    3: Config(3, _spec("r0.02_100x98_Z10000", 100, 98, 10000, 10, 8, 3, 18, 0.02, 3), 1, 500, 1, (0.3,),
              "rate-0.02 n=1e6, 1 frame, max 500 iterations, early stop on"),
    # config 4 is the code of config 3 (same seed) with 64 frames
    4: Config(4, _spec("r0.02_100x98_Z10000", 100, 98, 10000, 10, 8, 3, 18, 0.02, 3), 64, 500, 1, (0.3,),
              "batched throughput: config-3 code, 64 frames, max 500 iterations, early stop per frame"),
    5: Config(5, _spec("r0.05_100x95_Z10000", 100, 95, 10000, 10, 5, 3, 18, 0.05, 5), 32, 300, 1,
              (0.1, 0.3, 0.5, 0.7, 0.9, 1.1),
              "rate-0.05 n=1e6, 32 frames per point, 6 SNR points, max 300 iterations, early stop on"),
}


def scaled_spec(spec: CodeSpec, Z: int) -> CodeSpec:
    """Same base matrix (same seed), different lifting size: used for reduced-size parity cases."""
    return CodeSpec(f"{spec.name.rsplit('_Z', 1)[0]}_Z{Z}", spec.nb, spec.mb, Z, spec.n_core, spec.top_rows,
                    spec.top_deg, spec.low_deg, spec.rate, spec.seed)


def sigma_for_gap(rate: float, gap_db: float) -> float:
    """Noise std-dev `gap_db` dB above the BIAWGN capacity threshold of `rate`: sigma^2 = sigma*^2 10^(-gap/10)."""
    return SIGMA_STAR[rate] * 10.0 ** (-gap_db / 20.0)


def make_base_matrix(spec: CodeSpec) -> np.ndarray:
    """Deterministic base matrix of circulant shifts, int32 [mb][nb], -1 = zero block.

    The *structure* (which cells are non-zero) depends only on spec.seed, the shifts on (spec.seed, Z), so that
    `scaled_spec` keeps the graph and only re-draws shifts.
    """
    rng = np.random.default_rng(spec.seed)
    nb, mb, nc = spec.nb, spec.mb, spec.n_core
    n_low = mb - spec.top_rows
    assert nb - nc == n_low, "one degree-1 column per lower row"
    assert nc * spec.low_deg == 2 * n_low, "every lower row receives exactly 2 core edges"
    mask = np.zeros((mb, nb), dtype=bool)

    # top part: top_deg distinct random rows per core column; re-draw until every top row has degree >= 2 (S11)
    while True:
        top = np.zeros((spec.top_rows, nc), dtype=bool)
        for c in range(nc):
            top[rng.choice(spec.top_rows, size=spec.top_deg, replace=False), c] = True
        if top.sum(axis=1).min() >= 2:
            break
    mask[:spec.top_rows, :nc] = top

    # lower part: shuffle the multiset {each lower row x 2}, deal low_deg sockets per core column, re-draw until
    # every column's rows are distinct (S14)
    sockets = np.repeat(np.arange(n_low), 2)
    while True:
        perm = rng.permutation(sockets).reshape(nc, spec.low_deg)
        if all(len(set(perm[c])) == spec.low_deg for c in range(nc)):
            break
    for c in range(nc):
        mask[spec.top_rows + perm[c], c] = True

    base = np.full((mb, nb), -1, dtype=np.int32)
    srng = np.random.default_rng([spec.seed, spec.Z])
    base[mask] = srng.integers(0, spec.Z, size=int(mask.sum()), dtype=np.int32)
    # degree-1 diagonal, unshifted
    for j in range(nc, nb):
        base[j - nc + spec.top_rows, j] = 0
    return base


def syndrome_of(base_shifts: np.ndarray, Z: int, x: np.ndarray) -> np.ndarray:
    """s = H x mod 2 for x uint8 [..., nb*Z] by the lifting rule of P:324: s[R*Z+r] ^= x[C*Z + (r+p) mod Z]."""
    mb, nb = base_shifts.shape
    xs = x.reshape(x.shape[:-1] + (nb, Z))
    s = np.zeros(x.shape[:-1] + (mb, Z), dtype=np.uint8)
    for R in range(mb):
        for C in np.nonzero(base_shifts[R] >= 0)[0]:
            s[..., R, :] ^= np.roll(xs[..., C, :], -int(base_shifts[R, C]), axis=-1)
    return s.reshape(x.shape[:-1] + (mb * Z,))


@dataclass
class Frames:
    x: np.ndarray          # uint8 [F][n] transmitted word
    syndrome: np.ndarray   # uint8 [F][m]
    llr: np.ndarray        # float32 [F][n]
    sigma: float


def make_frames(base_shifts: np.ndarray, Z: int, sigma: float, n_frames: int, seed_base: int,
                first_frame: int = 0) -> Frames:
    """Frames first_frame .. first_frame+n_frames-1; frame f depends only on (seed_base + f)."""
    mb, nb = base_shifts.shape
    n = nb * Z
    x = np.empty((n_frames, n), dtype=np.uint8)
    llr = np.empty((n_frames, n), dtype=np.float32)
    for k in range(n_frames):
        rng = np.random.default_rng(seed_base + first_frame + k)
        x[k] = rng.integers(0, 2, size=n, dtype=np.uint8)
        y = (1.0 - 2.0 * x[k].astype(np.float64)) + sigma * rng.standard_normal(n)
        llr[k] = (2.0 * y / (sigma * sigma)).astype(np.float32)
    return Frames(x=x, syndrome=syndrome_of(base_shifts, Z, x), llr=llr, sigma=sigma)


def frame_seed_base(cfg_index: int, snr_point: int = 0) -> int:
    return FRAME_SEED_BASE + 1000 * cfg_index + 100 * snr_point


def make_config(cfg_index: int, snr_point: int = 0, n_frames: int | None = None, Z: int | None = None,
                first_frame: int = 0):
    """(config, base_shifts, Z, frames) for a BASELINE.json config; Z / n_frames override for reduced cases."""
    cfg = CONFIGS[cfg_index]
    spec = cfg.code if Z is None else scaled_spec(cfg.code, Z)
    base = make_base_matrix(spec)
    sigma = sigma_for_gap(spec.rate, cfg.gaps_db[snr_point])
    nf = cfg.n_frames if n_frames is None else n_frames
    frames = make_frames(base, spec.Z, sigma, nf, frame_seed_base(cfg_index, snr_point), first_frame)
    return cfg, base, spec.Z, frames


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-1: the paper's own rate-0.02 multi-edge ensemble, lifted by q.
# Three edge types.  Variable nodes (fractions of nb base columns, Omega):  9/400 with 2 type-1 + 57 type-2
# sockets, 7/400 with 3 type-1 + 57 type-2, 24/25 with one type-3 socket (the degree-1 diagonal).  Check nodes
# (Psi): 3/5 with 2 type-2 + 1 type-3, 9/25 with 3 type-2 + 1 type-3, and the "top" checks with type-1
# sockets only.  Reading G1: as printed, Psi's type-1 coefficients (3/320 on x1^3, 17/1600 on x1^7) do not
# balance the type-1 sockets of Omega (97.5 vs 102.5 per 1000 columns); swapped (17/1600 on x1^3, 3/320 on x1^7) they do,
# and the total edge count matches P:499.  For block lengths where those fractions are not integers the numbers of
# degree-3 and degree-7 top checks are the integers (a, b) with 3a + 7b = type-1 sockets and a + b closest to nb/50,
# which is what the paper's q = 50 code does (n = 1e6, rate 0.01995 instead of 0.02).
@dataclass(frozen=True)
class EnsembleSpec:
    nb: int                # base columns (n / q)
    q: int                 # expansion factor (Z)
    n_core2: int           # columns with 2 type-1 + 57 type-2 sockets
    n_core3: int           # columns with 3 type-1 + 57 type-2 sockets
    n_d1: int              # degree-1 columns
    rows_t3: int           # top checks of degree 3 (type 1 only)
    rows_t7: int           # top checks of degree 7
    rows_l2: int           # lower checks with 2 type-2 sockets (+ 1 type-3)
    rows_l3: int           # lower checks with 3 type-2 sockets (+ 1 type-3)
    seed: int

    @property
    def mb(self) -> int:
        return self.rows_t3 + self.rows_t7 + self.rows_l2 + self.rows_l3

    @property
    def n(self) -> int:
        return self.nb * self.q

    @property
    def m(self) -> int:
        return self.mb * self.q

    @property
    def base_edges(self) -> int:
        return (2 * self.n_core2 + 3 * self.n_core3) + 57 * (self.n_core2 + self.n_core3) + self.n_d1


PAPER_ENSEMBLE_SEED = 17020776000


def paper_ensemble_spec(nb: int, q: int, seed: int = PAPER_ENSEMBLE_SEED) -> EnsembleSpec:
    """Node counts of the ensemble at nb base columns (nb must be a multiple of 400 so that Omega's fractions and the
    lower-check fractions 3/5, 9/25 are integers)."""
    if nb % 400:
        raise ValueError("nb must be a multiple of 400")
    c2, c3, d1 = 9 * nb // 400, 7 * nb // 400, 24 * nb // 25
    l2, l3 = 3 * nb // 5, 9 * nb // 25
    assert l2 + l3 == d1 and 2 * l2 + 3 * l3 == 57 * (c2 + c3)
    s1 = 2 * c2 + 3 * c3                                    # type-1 sockets on the variable side
    best = None
    for b in range(s1 // 7 + 1):
        if (s1 - 7 * b) % 3 == 0:
            a = (s1 - 7 * b) // 3
            score = (abs((a + b) - nb / 50.0), abs(b - 3.0 * nb / 320.0))
            if best is None or score < best[0]:
                best = (score, a, b)
    if best is None:
        raise ValueError("type-1 sockets cannot be split into checks of degree 3 and 7")
    return EnsembleSpec(nb, q, c2, c3, d1, best[1], best[2], l2, l3, seed)


def _match_sockets(rng: np.random.Generator, vn_sockets: np.ndarray, cn_sockets: np.ndarray):
    """Random edge-type matching: pair every variable socket with a check socket of the same type,
    uniformly at random, then repair parallel edges (two edges between one column and one row cannot be one
    circulant) by swapping the offending variable socket with a random other one until none is left."""
    assert len(vn_sockets) == len(cn_sockets)
    cols = rng.permutation(vn_sockets)
    rows = cn_sockets.copy()
    for _ in range(10000):
        key = rows.astype(np.int64) * (int(cols.max()) + 1) + cols
        order = np.argsort(key, kind="stable")
        dup = order[1:][key[order][1:] == key[order][:-1]]
        if len(dup) == 0:
            return rows, cols
        other = rng.integers(0, len(cols), size=len(dup))
        for a, b in zip(dup, other):
            cols[a], cols[b] = cols[b], cols[a]
    raise RuntimeError("could not remove parallel edges")


def make_paper_ensemble(spec: EnsembleSpec):
    """Base graph of the paper's ensemble as the non-zero blocks (rows, cols, shifts), int32 arrays of length
    spec.base_edges, plus (mb, nb).  Columns: the n_core2 + n_core3 core columns first, then the degree-1 diagonal;
    rows: top checks (degree 3, then degree 7) first, then the lower checks (2, then 3 type-2 sockets); degree-1 column
    nc + r is the unshifted identity on lower row n_top + r (Fig. 11).  Shifts of all other blocks are
    uniform in [0, q).  The structure depends on spec.seed only, the shifts on (spec.seed, q)."""
    rng = np.random.default_rng(spec.seed)
    nc = spec.n_core2 + spec.n_core3
    n_top = spec.rows_t3 + spec.rows_t7
    n_low = spec.rows_l2 + spec.rows_l3
    deg1 = np.concatenate([np.full(spec.n_core2, 2), np.full(spec.n_core3, 3)])
    vn1 = np.repeat(np.arange(nc), deg1)
    cn1 = np.repeat(np.arange(n_top), np.concatenate([np.full(spec.rows_t3, 3), np.full(spec.rows_t7, 7)]))
    r1, c1 = _match_sockets(rng, vn1, cn1)
    vn2 = np.repeat(np.arange(nc), 57)
    cn2 = n_top + np.repeat(np.arange(n_low), np.concatenate([np.full(spec.rows_l2, 2), np.full(spec.rows_l3, 3)]))
    r2, c2 = _match_sockets(rng, vn2, cn2)
    rows = np.concatenate([r1, r2, n_top + np.arange(n_low)]).astype(np.int32)
    cols = np.concatenate([c1, c2, nc + np.arange(n_low)]).astype(np.int32)
    srng = np.random.default_rng([spec.seed, spec.q])
    shifts = np.concatenate([srng.integers(0, spec.q, size=len(r1) + len(r2)), np.zeros(n_low, dtype=np.int64)])
    return rows, cols, shifts.astype(np.int32), spec.mb, spec.nb


def syndrome_of_sparse(rows, cols, shifts, mb: int, nb: int, Z: int, x: np.ndarray) -> np.ndarray:
    """s = H x mod 2 for x uint8 [..., nb*Z], H given by its non-zero blocks (lifting rule P:324)."""
    xs = x.reshape(x.shape[:-1] + (nb, Z))
    s = np.zeros(x.shape[:-1] + (mb, Z), dtype=np.uint8)
    idx = (np.arange(Z)[None, :] + np.asarray(shifts)[:, None]) % Z          # [entries][Z]: (r + p) mod Z
    for k in range(len(rows)):
        s[..., rows[k], :] ^= xs[..., cols[k], :][..., idx[k]]
    return s.reshape(x.shape[:-1] + (mb * Z,))


def make_frames_sparse(rows, cols, shifts, mb: int, nb: int, Z: int, sigma: float, n_frames: int,
                       seed_base: int) -> Frames:
    """As make_frames, for a code given by its non-zero blocks."""
    n = nb * Z
    x = np.empty((n_frames, n), dtype=np.uint8)
    llr = np.empty((n_frames, n), dtype=np.float32)
    for k in range(n_frames):
        rng = np.random.default_rng(seed_base + k)
        x[k] = rng.integers(0, 2, size=n, dtype=np.uint8)
        y = (1.0 - 2.0 * x[k].astype(np.float64)) + sigma * rng.standard_normal(n)
        llr[k] = (2.0 * y / (sigma * sigma)).astype(np.float32)
    return Frames(x=x, syndrome=syndrome_of_sparse(rows, cols, shifts, mb, nb, Z, x), llr=llr, sigma=sigma)


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-2: the paper's second operating point -- rate 1/10, n = 2^20, q = 512, SNR 0.161, 100 iterations
# (Table IV).  The paper does NOT print that code's degree distribution (refs [25], [39]); this is a labelled
# STAND-IN with the shape of BASELINE.json's rate-0.1 configs at the paper's base-graph size: nb/5 core columns with 3
# edges into nb/10 top checks and 7 or 8 edges into the lower checks (each lower check: 2 core edges + 1 degree-1
# column on the unshifted diagonal).  It measures the decoder on that SIZE and lifting factor, nothing else.
def make_rate10_standin(nb: int = 2048, q: int = 512, seed: int = 17020777000):
    """Non-zero blocks (rows, cols, shifts, mb, nb) of the stand-in; structure from seed, shifts from (seed, q)."""
    rng = np.random.default_rng(seed)
    nc = (nb + 2) // 5
    n_top = nb // 10
    n_low = nb - nc
    mb = n_top + n_low
    while True:                                            # 3 distinct top checks per core column, every top check >= 2
        top = np.stack([rng.choice(n_top, size=3, replace=False) for _ in range(nc)])
        if np.bincount(top.ravel(), minlength=n_top).min() >= 2:
            break
    r1, c1 = top.ravel(), np.repeat(np.arange(nc), 3)
    sockets = np.repeat(np.arange(n_low), 2)               # every lower check receives exactly 2 core edges
    share = np.full(nc, len(sockets) // nc)
    share[: len(sockets) - share.sum()] += 1               # 8, 8, ..., 7: dealt in column order
    vn2 = np.repeat(np.arange(nc), share)
    r2, c2 = _match_sockets(rng, vn2, n_top + sockets)
    rows = np.concatenate([r1, r2, n_top + np.arange(n_low)]).astype(np.int32)
    cols = np.concatenate([c1, c2, nc + np.arange(n_low)]).astype(np.int32)
    srng = np.random.default_rng([seed, q])
    shifts = np.concatenate([srng.integers(0, q, size=len(r1) + len(r2)), np.zeros(n_low, dtype=np.int64)])
    return rows, cols, shifts.astype(np.int32), mb, nb
