"""Seeded synthetic workloads (BASELINE.json `configs[0..4]`).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests / bench.
It holds none of the method's arithmetic: it draws a matrix, plants trend biclusters by sorting
values, injects NaN, and draws a population.  It imports numpy only (no torch, no CUDA library,
no oracle).

The matrices stand in for the paper's GEO datasets (Table 1, lines 69-75: GDS1490,
GSE65194, GSE84493), which are not available offline: shapes, value ranges and row counts follow
them (expression values ~N(0,1), methylation beta values in [0,1], 10^4 .. 4.4*10^5 rows) and
BASELINE.json fixes the rest.  Recipe (fixed order of draws, `rng = default_rng([0, index])`):

 1. matrix: U[0,1) / N(0,1) / Beta(.5,.5) as float32, row-major [rows][cols];
 2. per bicluster: its size, then row sets (disjoint across biclusters, drawn without
    replacement), then an ordered column subset;
 3. planting: the row's existing values at the planted columns are sorted ascending and written
    back in planted order (the marginal distribution is kept).  `exact` workloads (C1) re-draw
    rows with ties so planted rows are STRICTLY increasing, use disjoint column sets, and force
    every non-member row to descend between the first two planted columns, so that the planted
    row set is exactly the set of rows following the planted order;
 4. NaN: `rng.random(float32) < nan_rate` in chunks of 2^20 rows;
 5. population: for every bicluster its planted chromosome and three order-preserving random
    sub-sequences of it (individuals with large counts, as in a converged GA), then uniformly
    random individuals: L uniform in the length range, L distinct columns in random order.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

MISSING_OFF = 0
MISSING_ON = 1

_NAN_CHUNK_ROWS = 1 << 20


@dataclass(frozen=True)
class WorkloadConfig:
    index: int
    name: str
    rows: int
    cols: int
    dist: str                      # "uniform" | "normal" | "beta"
    n_bic: int
    bic_rows: Tuple[int, int]      # inclusive range of planted rows per bicluster
    bic_cols: Tuple[int, int]      # inclusive range of planted columns per bicluster
    nan_rate: float
    missing_mode: int
    n_ind: int
    len_range: Tuple[int, int]     # inclusive chromosome length range
    exact: bool = False            # planted row set is exactly recoverable (C1)


CONFIGS: Tuple[WorkloadConfig, ...] = (
    WorkloadConfig(0, "C1-tiny", 200, 20, "uniform", 2, (30, 30), (5, 5), 0.0, MISSING_OFF,
                   64, (2, 6), exact=True),
    WorkloadConfig(1, "C2-expression-like", 10_000, 100, "normal", 5, (100, 500), (4, 10), 0.02,
                   MISSING_ON, 1_600, (2, 10)),
    WorkloadConfig(2, "C3-beyond-old-grid-limit", 100_000, 50, "normal", 10, (200, 2_000), (3, 8),
                   0.0, MISSING_OFF, 1_600, (2, 12)),
    WorkloadConfig(3, "C4-methylation-like", 436_444, 64, "beta", 20, (500, 5_000), (4, 10), 0.01,
                   MISSING_ON, 1_600, (2, 20)),
    WorkloadConfig(4, "C5-stress", 16_777_216, 32, "uniform", 50, (1_000, 50_000), (3, 8), 0.005,
                   MISSING_ON, 4_096, (2, 16)),
)

# stand-ins with the shapes of the paper's own datasets (Table 1, lines
# 73-75: GDS1490 12,483 x 150, GSE65194 54,675 x 178, GSE84493 436,444 x 310) and its typical population
# (1,600).  Wider than 127 columns: no rank tiles; a float tile of all columns no longer
# double-buffers in shared memory at 310 columns.  `make_workload(5..7)`; not BASELINE.json configs.
PAPER_SHAPES: Tuple[WorkloadConfig, ...] = (
    WorkloadConfig(5, "P1-GDS1490-shaped", 12_483, 150, "normal", 5, (100, 500), (4, 10), 0.0,
                   MISSING_OFF, 1_600, (2, 20)),
    WorkloadConfig(6, "P2-GSE65194-shaped", 54_675, 178, "normal", 10, (200, 2_000), (4, 10), 0.01,
                   MISSING_ON, 1_600, (2, 20)),
    WorkloadConfig(7, "P3-GSE84493-shaped", 436_444, 310, "beta", 20, (500, 5_000), (4, 10), 0.01,
                   MISSING_ON, 1_600, (2, 20)),
)


@dataclass
class Bicluster:
    rows: np.ndarray        # sorted int64 row indices
    order: np.ndarray       # int32 column ids in planted (ascending-value) order
    clean_rows: np.ndarray  # subset of `rows` with no injected NaN in the planted columns


@dataclass
class Workload:
    cfg: WorkloadConfig
    rows: int
    cols: int
    missing_mode: int
    matrix: np.ndarray      # float32 [rows][cols], C-contiguous (row-major)
    offsets: np.ndarray     # int32 [n_ind+1]
    col_ids: np.ndarray     # int32 [offsets[-1]]
    planted: List[Bicluster] = field(default_factory=list)
    planted_individuals: List[Tuple[int, int]] = field(default_factory=list)  # (individual, bicluster)

    @property
    def n_ind(self) -> int:
        return int(self.offsets.size - 1)

    @property
    def lengths(self) -> np.ndarray:
        return np.diff(self.offsets)

    @property
    def comparisons(self) -> int:
        """Nominal row-pair comparisons of one whole-population evaluation (BASELINE.json metric)."""
        return int(self.rows) * int(np.maximum(self.lengths - 1, 0).sum())

    @property
    def visits(self) -> int:
        """Nominal (row, column-visit) operand fetches: rows * sum(L)."""
        return int(self.rows) * int(self.lengths.sum())


def _draw_matrix(rng: np.random.Generator, dist: str, rows: int, cols: int) -> np.ndarray:
    if dist == "uniform":
        return rng.random((rows, cols), dtype=np.float32)
    if dist == "normal":
        return rng.standard_normal((rows, cols), dtype=np.float32)
    if dist == "beta":
        return rng.beta(0.5, 0.5, size=(rows, cols)).astype(np.float32)
    raise ValueError(f"unknown distribution {dist!r}")


def make_population(rng: np.random.Generator, cols: int, n_ind: int, len_range: Tuple[int, int],
                    seeds: Optional[List[np.ndarray]] = None):
    """CSR population: `seeds` (ordered column lists) first, then uniformly random individuals."""
    lo, hi = len_range
    hi = min(hi, cols)
    lo = min(lo, hi)
    chrom: List[np.ndarray] = []
    for s in (seeds or []):
        if len(chrom) >= n_ind:
            break
        chrom.append(np.asarray(s, dtype=np.int32))
    while len(chrom) < n_ind:
        L = int(rng.integers(lo, hi + 1))
        chrom.append(rng.choice(cols, size=L, replace=False).astype(np.int32))
    lengths = np.array([c.size for c in chrom], dtype=np.int64)
    offsets = np.zeros(n_ind + 1, dtype=np.int32)
    offsets[1:] = np.cumsum(lengths)
    col_ids = np.concatenate(chrom).astype(np.int32) if chrom else np.zeros(0, dtype=np.int32)
    return offsets, col_ids


def make_workload(index: int, rows: Optional[int] = None, n_ind: Optional[int] = None) -> Workload:
    """Build workload C(index+1) (index 0..4) or a paper-shaped stand-in (index 5..7).  `rows` / `n_ind`
    resize it (same recipe) for parity tests."""
    cfg = (CONFIGS + PAPER_SHAPES)[index]
    rows = int(cfg.rows if rows is None else rows)
    n_ind = int(cfg.n_ind if n_ind is None else n_ind)
    cols = cfg.cols
    rng = np.random.default_rng([0, cfg.index])

    # 1. matrix
    M = _draw_matrix(rng, cfg.dist, rows, cols)

    # 2. bicluster shapes, disjoint row sets, ordered column subsets
    cap = max(2, rows // (2 * cfg.n_bic))
    n_rows_b = [min(int(rng.integers(cfg.bic_rows[0], cfg.bic_rows[1] + 1)), cap)
                for _ in range(cfg.n_bic)]
    n_cols_b = [min(int(rng.integers(cfg.bic_cols[0], cfg.bic_cols[1] + 1)), cols)
                for _ in range(cfg.n_bic)]
    all_rows = rng.choice(rows, size=sum(n_rows_b), replace=False).astype(np.int64)
    row_sets, pos = [], 0
    for nr in n_rows_b:
        row_sets.append(np.sort(all_rows[pos:pos + nr]))
        pos += nr
    if cfg.exact:
        if sum(n_cols_b) > cols:
            raise ValueError("exact workloads need disjoint planted column sets")
        perm = rng.permutation(cols).astype(np.int32)
        orders, pos = [], 0
        for nc in n_cols_b:
            orders.append(perm[pos:pos + nc].copy())
            pos += nc
    else:
        orders = [rng.choice(cols, size=nc, replace=False).astype(np.int32) for nc in n_cols_b]

    # 3. planting
    for rs, order in zip(row_sets, orders):
        sub = np.sort(M[np.ix_(rs, order)], axis=1)
        if cfg.exact:
            while True:
                tied = (np.diff(sub, axis=1) <= 0).any(axis=1)
                if not tied.any():
                    break
                sub[tied] = np.sort(_draw_matrix(rng, cfg.dist, int(tied.sum()), order.size), axis=1)
        M[np.ix_(rs, order)] = sub
    if cfg.exact:
        for rs, order in zip(row_sets, orders):
            others = np.setdiff1d(np.arange(rows, dtype=np.int64), rs)
            a = M[others, order[0]].copy()
            b = M[others, order[1]].copy()
            swap = b >= a
            M[others[swap], order[0]] = b[swap]
            M[others[swap], order[1]] = a[swap]
            eq = M[others, order[1]] == M[others, order[0]]
            if eq.any():
                M[others[eq], order[1]] = np.nextafter(M[others[eq], order[1]], np.float32(-np.inf))

    # 4. NaN injection
    if cfg.nan_rate > 0.0:
        p = np.float32(cfg.nan_rate)
        for r0 in range(0, rows, _NAN_CHUNK_ROWS):
            r1 = min(rows, r0 + _NAN_CHUNK_ROWS)
            hit = rng.random((r1 - r0, cols), dtype=np.float32) < p
            M[r0:r1][hit] = np.float32(np.nan)
    planted = []
    for rs, order in zip(row_sets, orders):
        has_nan = np.isnan(M[np.ix_(rs, order)]).any(axis=1)
        planted.append(Bicluster(rows=rs, order=order, clean_rows=rs[~has_nan]))

    # 5. population
    seeds: List[np.ndarray] = []
    planted_individuals: List[Tuple[int, int]] = []
    budget = max(1, n_ind // 4)
    for b, bic in enumerate(planted):
        if len(seeds) >= budget:
            break
        planted_individuals.append((len(seeds), b))
        seeds.append(bic.order.copy())
        for _ in range(3):
            if len(seeds) >= budget or bic.order.size < 3:
                break
            L = int(rng.integers(2, bic.order.size))
            keep = np.sort(rng.choice(bic.order.size, size=L, replace=False))
            seeds.append(bic.order[keep].copy())
    offsets, col_ids = make_population(rng, cols, n_ind, cfg.len_range, seeds)

    return Workload(cfg=cfg, rows=rows, cols=cols, missing_mode=cfg.missing_mode,
                    matrix=np.ascontiguousarray(M), offsets=offsets, col_ids=col_ids,
                    planted=planted, planted_individuals=planted_individuals)


def random_case(seed: int, rows: int, cols: int, n_ind: int, len_range=(0, 6), nan_rate=0.0,
                ties: bool = False, distinct: bool = True):
    """Small free-form case for property tests: (matrix, offsets, col_ids).

    `ties=True` quantises values to a few levels (many equal pairs); `distinct=False` allows
    repeated columns inside a chromosome.
    """
    rng = np.random.default_rng([1, seed])
    M = rng.standard_normal((rows, cols), dtype=np.float32)
    if ties:
        M = np.round(M * 2.0).astype(np.float32) / np.float32(2.0)
    if nan_rate > 0:
        M[rng.random((rows, cols)) < nan_rate] = np.float32(np.nan)
    lo, hi = len_range
    chrom = []
    for _ in range(n_ind):
        L = int(rng.integers(lo, hi + 1))
        if distinct:
            L = min(L, cols)
            chrom.append(rng.choice(cols, size=L, replace=False).astype(np.int32))
        else:
            chrom.append(rng.integers(0, cols, size=L).astype(np.int32))
    offsets = np.zeros(n_ind + 1, dtype=np.int32)
    offsets[1:] = np.cumsum([c.size for c in chrom])
    col_ids = (np.concatenate(chrom) if chrom else np.zeros(0)).astype(np.int32)
    return np.ascontiguousarray(M), offsets, col_ids


def draw_matrix(rng: np.random.Generator, dist: str, rows: int, cols: int) -> np.ndarray:
    """A rows x cols float32 matrix of the named distribution ("uniform", "normal", "beta"): the draw behind the
    C1-C5 / P1-P3 workloads, for callers that need more rows of the same kind (bench.py's weak-scaling ranks)."""
    return _draw_matrix(rng, dist, rows, cols)


def big_matrix(seed: int, rows: int, cols: int, levels: int = 8, n_nan: int = 0, nan_rows=()) -> np.ndarray:
    """A matrix for the index-width tests (up to 2^31-1 rows): float32 [rows][cols] filled chunk by
    chunk into ONE preallocated array (the host never holds a second copy), values = small integers 0..levels-1 (many
    ties, so that both orders of a column pair match on a good share of the rows), `n_nan` cells at seeded random
    positions and one cell in each of `nan_rows` set to NaN."""
    rng = np.random.default_rng([9, seed])
    m = np.empty((rows, cols), dtype=np.float32)
    step = max(1, (1 << 26) // cols)
    for r0 in range(0, rows, step):
        blk = m[r0:r0 + step]
        blk[...] = rng.integers(0, levels, size=blk.shape, dtype=np.int8)
    if n_nan:
        m[rng.integers(0, rows, size=n_nan), rng.integers(0, cols, size=n_nan)] = np.float32(np.nan)
    for i, r in enumerate(nan_rows):
        m[r, i % cols] = np.float32(np.nan)
    return m
