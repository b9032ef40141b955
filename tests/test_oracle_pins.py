"""Pins for the CPU oracle (oracle/ebic_oracle.c) against things other than itself.

The paper prints no worked example, so the pins are: hand-enumerated
fixtures (tests/golden/), exact planted recovery, invariants, identities, a closed form, special
matrices, a pure-Python brute force and an independent numpy restatement -- SURVEY.md section
8(c), pins 1-9.  Each is chosen so that a plausible mistake (dropped term, wrong sign or index,
transposed operand, wrong NaN rule, flush-to-zero, off-by-one in the bit layout) fails it.
"""
from __future__ import annotations

import itertools
import math

import numpy as np
import pytest

from conftest import (brute_force_ok, csr, golden_names, load_golden, mask_to_bits, numpy_ok)
from paper_1807_09932_b200 import workloads as W

ON, OFF = 1, 0


def _modes(tag):
    return {"ON": [ON], "OFF": [OFF], "BOTH": [ON, OFF]}[tag]


# ---------------------------------------------------------------- pin 1: hand-enumerated fixtures
@pytest.mark.parametrize("name", golden_names())
def test_golden_fixture(oracle_mod, name):
    m, cases = load_golden(name)
    for case in cases:
        off, ids = csr([case["ids"]])
        want = np.array([ch == "1" for ch in case["mask"]])
        for mode in _modes(case["mode"]):
            st, counts = oracle_mod.eval_fitness(m, mode, off, ids)
            assert st == oracle_mod.OK
            assert int(counts[0]) == case["count"], (name, case, mode)
            st, masks, c2 = oracle_mod.extract_rows(m, mode, off, ids, [0])
            assert st == oracle_mod.OK
            assert int(c2[0]) == case["count"]
            assert (mask_to_bits(masks[0], m.shape[0]) == want).all(), (name, case, mode)
            # the two independent restatements agree with the hand-typed answer as well
            assert (brute_force_ok(m, case["ids"], mode == ON) == want).all()
            assert (numpy_ok(m, case["ids"], mode == ON) == want).all()


def test_golden_whole_population_at_once(oracle_mod):
    """All cases of a fixture as ONE population: catches offset / indexing slips across individuals."""
    for name in golden_names():
        m, cases = load_golden(name)
        for mode in (ON, OFF):
            sel = [c for c in cases if mode in _modes(c["mode"])]
            off, ids = csr([c["ids"] for c in sel])
            st, counts = oracle_mod.eval_fitness(m, mode, off, ids)
            assert st == 0
            assert counts.tolist() == [c["count"] for c in sel]
            chosen = list(range(len(sel)))[::-1]
            st, masks, c2 = oracle_mod.extract_rows(m, mode, off, ids, chosen)
            assert c2.tolist() == [sel[j]["count"] for j in chosen]
            for slot, j in enumerate(chosen):
                want = np.array([ch == "1" for ch in sel[j]["mask"]])
                assert (mask_to_bits(masks[slot], m.shape[0]) == want).all()


def test_nan_bit_patterns(oracle_mod):
    """R3: every NaN encoding is 'missing' (quiet, signalling, negative, payloads); inf is not."""
    pats = np.array([0x7fc00000, 0xffc00000, 0x7f800001, 0xff800001, 0x7fffffff, 0x7fa00000,
                     0x7f800000, 0xff800000, 0x00000000, 0x80000000], dtype=np.uint32)
    col0 = pats.view(np.float32)
    m = np.stack([col0, np.zeros_like(col0)], axis=1).copy()
    off, ids = csr([[0], [0, 0], [1, 0]])
    st, counts = oracle_mod.eval_fitness(m, ON, off, ids)
    # rows 0-5 are NaN; rows 6,7 (+-inf), 8,9 (+-0) are values.  [1,0]: col0 >= 0.0 -> +inf, +0, -0
    assert counts.tolist() == [4, 4, 3]
    st, counts = oracle_mod.eval_fitness(m, OFF, off, ids)
    assert counts.tolist() == [10, 4, 3]


# ---------------------------------------------------------------- pin 2: planted recovery
def test_planted_recovery_exact_c1(oracle_mod):
    w = W.make_workload(0)
    assert (w.rows, w.cols, w.n_ind) == (200, 20, 64)
    assert len(w.planted) == 2 and all(b.rows.size == 30 and b.order.size == 5 for b in w.planted)
    chosen = [k for k, _ in w.planted_individuals]
    st, masks, counts = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    assert st == 0
    for slot, (k, b) in enumerate(w.planted_individuals):
        got = np.flatnonzero(mask_to_bits(masks[slot], w.rows))
        assert got.tolist() == w.planted[b].rows.tolist()      # EXACTLY the planted rows
        assert int(counts[slot]) == 30
    st, all_counts = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    for k, b in w.planted_individuals:
        assert int(all_counts[k]) == 30
        # the sub-sequences that follow a planted chromosome keep all its rows
        for j in range(k + 1, k + 4):
            assert int(all_counts[j]) >= 30


@pytest.mark.parametrize("index,rows", [(1, 10_000), (3, 20_000)])
def test_planted_recovery_superset_with_nan(oracle_mod, index, rows):
    w = W.make_workload(index, rows=rows, n_ind=64)
    assert w.missing_mode == ON
    chosen = [k for k, _ in w.planted_individuals]
    st, masks, counts = oracle_mod.extract_rows(w.matrix, ON, w.offsets, w.col_ids, chosen)
    assert st == 0
    for slot, (k, b) in enumerate(w.planted_individuals):
        bits = mask_to_bits(masks[slot], w.rows)
        bic = w.planted[b]
        assert bits[bic.clean_rows].all()                      # every clean planted row is found
        dirty = np.setdiff1d(bic.rows, bic.clean_rows)
        assert not bits[dirty].any()                           # NaN in a planted column: not counted
        assert int(counts[slot]) == int(bits.sum())


# ---------------------------------------------------------------- pin 3: invariants
@pytest.mark.parametrize("seed,nan_rate,ties,distinct", [(0, 0.0, False, True), (1, 0.15, False, True),
                                                         (2, 0.1, True, True), (3, 0.1, True, False)])
def test_invariants(oracle_mod, seed, nan_rate, ties, distinct):
    rows, cols = 777, 9
    m, off, ids = W.random_case(seed, rows, cols, 120, (0, 6), nan_rate, ties, distinct)
    nonmissing = (~np.isnan(m)).sum(axis=0)
    res = {}
    for mode in (ON, OFF):
        st, counts = oracle_mod.eval_fitness(m, mode, off, ids)
        assert st == 0
        st, masks, c2 = oracle_mod.extract_rows(m, mode, off, ids, np.arange(off.size - 1))
        assert (counts == c2).all()
        for k in range(off.size - 1):
            chrom = ids[off[k]:off[k + 1]]
            bits = mask_to_bits(masks[k], rows)
            assert int(bits.sum()) == int(counts[k])           # popcount(mask) == count
            assert (bits == numpy_ok(m, chrom, mode == ON)).all()
            if chrom.size == 0:
                assert counts[k] == rows
            if chrom.size == 1:
                assert counts[k] == (nonmissing[chrom[0]] if mode == ON else rows)
            if chrom.size >= 2 or mode == ON:
                if chrom.size:
                    assert counts[k] <= nonmissing[chrom].min()
        res[mode] = counts
    # pin 4: ON and OFF differ only for L = 1 (reading R4)
    L = np.diff(off)
    assert (res[ON][L != 1] == res[OFF][L != 1]).all()


def test_subsequence_monotone(oracle_mod):
    """count(S) >= count(T) whenever S is a subsequence of T (prefix extension is a special case)."""
    rows, cols = 1500, 8
    m, _, _ = W.random_case(7, rows, cols, 1, (1, 1), 0.05, True, True)
    rng = np.random.default_rng(11)
    chroms = []
    for _ in range(60):
        T = rng.permutation(cols)[: int(rng.integers(2, 7))]
        keep = np.sort(rng.choice(T.size, size=int(rng.integers(0, T.size)), replace=False))
        chroms += [T.tolist(), T[keep].tolist(), T[:-1].tolist()]
    off, ids = csr(chroms)
    for mode in (ON, OFF):
        st, counts = oracle_mod.eval_fitness(m, mode, off, ids)
        c = counts.reshape(-1, 3)
        assert (c[:, 1] >= c[:, 0]).all() and (c[:, 2] >= c[:, 0]).all()


# ---------------------------------------------------------------- pin 5: reversal identity (L = 2)
def test_reversal_identity(oracle_mod):
    rows, cols = 2000, 6
    m, _, _ = W.random_case(5, rows, cols, 1, (1, 1), 0.1, True, True)
    pairs = [(a, b) for a in range(cols) for b in range(cols) if a != b]
    off, ids = csr([list(p) for p in pairs])
    for mode in (ON, OFF):
        st, counts = oracle_mod.eval_fitness(m, mode, off, ids)
        cnt = dict(zip(pairs, counts.tolist()))
        for a, b in pairs:
            both = ~np.isnan(m[:, a]) & ~np.isnan(m[:, b])
            equal = both & (m[:, a] == m[:, b])
            assert cnt[(a, b)] + cnt[(b, a)] == int(both.sum()) + int(equal.sum())


# ---------------------------------------------------------------- pin 7: permutation partition
def test_permutation_partition(oracle_mod):
    rows, cols = 600, 7
    m, _, _ = W.random_case(9, rows, cols, 1, (1, 1), 0.08, True, True)
    for subset in [(0, 1), (2, 4, 6), (1, 3, 5, 6), (0, 2, 3, 4, 5)]:
        perms = list(itertools.permutations(subset))
        off, ids = csr([list(p) for p in perms])
        st, counts = oracle_mod.eval_fitness(m, ON, off, ids)
        expect = 0
        for r in range(rows):
            vals = [float(m[r, c]) for c in subset]
            if any(math.isnan(v) for v in vals):
                continue
            groups = {}
            for v in vals:
                groups[v + 0.0] = groups.get(v + 0.0, 0) + 1     # -0.0 and +0.0 are one group
            expect += math.prod(math.factorial(g) for g in groups.values())
        assert int(counts.sum()) == expect


# ---------------------------------------------------------------- pin 6: closed form (statistical)
def test_binomial_closed_form(oracle_mod):
    """iid continuous rows, L distinct columns: P(ok) = (1-p)^L / L!  ->  count within 5 sigma."""
    rows, cols, p = 200_000, 12, 0.01
    rng = np.random.default_rng(2024)
    m = rng.standard_normal((rows, cols), dtype=np.float32)
    m[rng.random((rows, cols)) < p] = np.nan
    chroms = [rng.permutation(cols)[:L].tolist() for L in (2, 3, 4, 5) for _ in range(12)]
    off, ids = csr(chroms)
    st, counts = oracle_mod.eval_fitness(m, ON, off, ids)
    for chrom, c in zip(chroms, counts.tolist()):
        L = len(chrom)
        q = (1 - p) ** L / math.factorial(L)
        sigma = math.sqrt(rows * q * (1 - q))
        assert abs(c - rows * q) <= 5 * sigma, (chrom, c, rows * q, sigma)


# ---------------------------------------------------------------- pin 8: special matrices
def test_special_matrices(oracle_mod):
    rows, cols = 333, 6
    const = np.full((rows, cols), 2.5, dtype=np.float32)
    _, off, ids = W.random_case(4, rows, cols, 40, (0, 6), 0.0, False, False)
    for mode in (ON, OFF):
        st, counts = oracle_mod.eval_fitness(const, mode, off, ids)
        assert (counts == rows).all()
    inc = (np.arange(cols, dtype=np.float32)[None, :] + 10 * np.arange(rows, dtype=np.float32)[:, None])
    _, off, ids = W.random_case(6, rows, cols, 60, (2, 6), 0.0, False, True)
    st, counts = oracle_mod.eval_fitness(np.ascontiguousarray(inc), ON, off, ids)
    for k in range(off.size - 1):
        chrom = ids[off[k]:off[k + 1]]
        assert counts[k] == (rows if (np.diff(chrom) > 0).all() else 0)


# ---------------------------------------------------------------- pin 9 + brute force on random input
@pytest.mark.parametrize("seed", [21, 22, 23])
def test_numpy_and_bruteforce_agree(oracle_mod, seed):
    rows, cols = 131, 5
    m, off, ids = W.random_case(seed, rows, cols, 25, (0, 7), 0.2, True, False)
    for mode in (ON, OFF):
        st, masks, counts = oracle_mod.extract_rows(m, mode, off, ids, np.arange(off.size - 1))
        assert st == 0
        for k in range(off.size - 1):
            chrom = ids[off[k]:off[k + 1]].tolist()
            bits = mask_to_bits(masks[k], rows)
            assert (bits == brute_force_ok(m, chrom, mode == ON)).all()
            assert (bits == numpy_ok(m, chrom, mode == ON)).all()


# ---------------------------------------------------------------- bit layout, sizes, errors
@pytest.mark.parametrize("rows", [1, 63, 64, 65, 127, 128, 129, 200])
def test_mask_layout_and_tail(oracle_mod, rows):
    m = np.zeros((rows, 2), dtype=np.float32)
    m[:, 1] = -1.0
    hit = [r for r in (0, 1, 31, 32, 62, 63, 64, 65, 127, 128, rows - 1) if r < rows]
    m[hit, 1] = 1.0
    off, ids = csr([[0, 1]])
    st, masks, counts = oracle_mod.extract_rows(m, ON, off, ids, [0])
    assert masks.shape == (1, (rows + 63) // 64)
    assert int(counts[0]) == len(set(hit))
    for r in range(rows):
        word, bit = divmod(r, 64)
        assert bool((int(masks[0, word]) >> bit) & 1) == (r in hit)
    as_bytes = masks[0].view(np.uint8)                      # same layout viewed as bytes, LSB first
    for r in hit:
        assert (int(as_bytes[r // 8]) >> (r % 8)) & 1
    if rows % 64:
        assert int(masks[0, -1]) >> (rows % 64) == 0        # tail bits zero


def test_errors(oracle_mod):
    m, _, _ = W.random_case(3, 50, 4, 1)
    good = [[0, 1], [2], []]
    off, ids = csr(good + [[1, 4]])                         # 4 == cols: out of range
    st, counts = oracle_mod.eval_fitness(m, ON, off, ids)
    assert st == oracle_mod.ERR_BAD_COLUMN and counts[3] == 0
    st0, ref = oracle_mod.eval_fitness(m, ON, *csr(good))
    assert st0 == 0 and (counts[:3] == ref).all()           # valid individuals unaffected
    off, ids = csr(good + [[-1, 2]])
    assert oracle_mod.eval_fitness(m, ON, off, ids)[0] == oracle_mod.ERR_BAD_COLUMN
    st, masks, c = oracle_mod.extract_rows(m, ON, off, ids, [3, 0])
    assert st == oracle_mod.ERR_BAD_COLUMN and not masks[0].any() and c[0] == 0 and c[1] == ref[0]
    bad_off = np.array([0, 2, 1, 3], dtype=np.int32)        # offsets[2] < offsets[1]
    ids3 = np.array([0, 1, 2], dtype=np.int32)
    st, counts = oracle_mod.eval_fitness(m, ON, bad_off, ids3)
    assert st == oracle_mod.ERR_BAD_OFFSETS and counts[1] == 0
    both = np.array([0, 2, 1, 3], dtype=np.int32)
    st, counts = oracle_mod.eval_fitness(m, ON, both, np.array([0, 9, 2], dtype=np.int32))
    assert st == oracle_mod.ERR_BAD_OFFSETS                 # larger code wins
    with pytest.raises(Exception):
        oracle_mod.eval_fitness(m.reshape(-1), ON, off, ids)
    assert oracle_mod.eval_fitness(m, 7, *csr(good))[0] == oracle_mod.ERR_ARG
    st, masks, c = oracle_mod.extract_rows(m, ON, *csr(good), [3, 1, -1])   # 3, -1: no such individual
    assert st == oracle_mod.ERR_BAD_OFFSETS and not masks[0].any() and not masks[2].any()
    assert c.tolist() == [0, int(ref[1]), 0]
    off_long = np.array([0, 2, 5], dtype=np.int32)         # offsets[2] > n_ids == 3
    st, counts = oracle_mod.eval_fitness(m, ON, off_long, np.array([0, 1, 2], dtype=np.int32))
    assert st == oracle_mod.ERR_BAD_OFFSETS and counts[1] == 0 and counts[0] == ref[0]
    st, counts = oracle_mod.eval_fitness(m, ON, np.zeros(1, np.int32), np.zeros(0, np.int32))
    assert st == 0 and counts.size == 0


def test_thread_count_does_not_matter(oracle_mod):
    w = W.make_workload(1, rows=3000, n_ind=200)
    a = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids, n_threads=1)[1]
    b = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids, n_threads=0)[1]
    assert (a == b).all()
