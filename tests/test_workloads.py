"""The seeded generators: deterministic, right shapes, and hold none of the method's results."""
from __future__ import annotations

import numpy as np
import pytest

from paper_1807_09932_b200 import workloads as W


def test_config_table_matches_baseline_json():
    shapes = [(c.rows, c.cols, c.n_ind, c.len_range, c.nan_rate, c.n_bic) for c in W.CONFIGS]
    assert shapes == [(200, 20, 64, (2, 6), 0.0, 2),
                      (10_000, 100, 1_600, (2, 10), 0.02, 5),
                      (100_000, 50, 1_600, (2, 12), 0.0, 10),
                      (436_444, 64, 1_600, (2, 20), 0.01, 20),
                      (16_777_216, 32, 4_096, (2, 16), 0.005, 50)]
    assert [c.missing_mode for c in W.CONFIGS] == [0, 1, 0, 1, 1]


@pytest.mark.parametrize("index", [0, 1, 2])
def test_deterministic_and_well_formed(index):
    a = W.make_workload(index)
    b = W.make_workload(index)
    assert a.matrix.tobytes() == b.matrix.tobytes()
    assert (a.offsets == b.offsets).all() and (a.col_ids == b.col_ids).all()
    cfg = a.cfg
    assert a.matrix.dtype == np.float32 and a.matrix.flags.c_contiguous
    assert a.matrix.shape == (cfg.rows, cfg.cols)
    assert a.offsets.dtype == np.int32 and a.col_ids.dtype == np.int32
    assert a.offsets[0] == 0 and a.offsets[-1] == a.col_ids.size and a.n_ind == cfg.n_ind
    L = a.lengths
    assert L.min() >= 2 and L.max() <= max(cfg.len_range[1], cfg.bic_cols[1])
    assert a.col_ids.min() >= 0 and a.col_ids.max() < cfg.cols
    for k in range(a.n_ind):                                   # distinct columns per chromosome
        c = a.col_ids[a.offsets[k]:a.offsets[k + 1]]
        assert np.unique(c).size == c.size
    nan_frac = np.isnan(a.matrix).mean()
    assert abs(nan_frac - cfg.nan_rate) < 0.002
    all_rows = np.concatenate([p.rows for p in a.planted])
    assert np.unique(all_rows).size == all_rows.size           # disjoint planted row sets
    assert a.comparisons == cfg.rows * int((L - 1).sum())


def test_scaled_down_variant_keeps_recipe():
    w = W.make_workload(4, rows=5000, n_ind=100)
    assert w.matrix.shape == (5000, 32) and w.n_ind == 100
    assert len(w.planted) == 50 and all(p.rows.size >= 2 for p in w.planted)


def test_paper_shaped_configs():
    """PAPER.md Table 1 (lines 73-75): the three dataset shapes; population 1,600."""
    assert [(c.index, c.rows, c.cols, c.n_ind) for c in W.PAPER_SHAPES] == [
        (5, 12_483, 150, 1_600), (6, 54_675, 178, 1_600), (7, 436_444, 310, 1_600)]
    w = W.make_workload(5, rows=2_000, n_ind=50)
    assert w.matrix.shape == (2_000, 150) and w.n_ind == 50 and w.col_ids.max() < 150
