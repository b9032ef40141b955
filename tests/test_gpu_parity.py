"""Parity of the CUDA path (through the C ABI, via the thin binding) against the CPU oracle.

Bar: bit-exact (integer counts and bitmasks from exact float32 comparisons; tolerance 0).
Every fitness kernel (DIRECT, TILED_F32, RANK8, PAIRBITS, UNION_F32, PREFIX, PAIRTILE) is compared with the oracle on the same seeded
inputs.  All tests here need the B200.
"""
from __future__ import annotations

import numpy as np
import pytest

from conftest import csr, golden_names, load_golden, mask_to_bits
from paper_1807_09932_b200 import workloads as W

pytestmark = pytest.mark.gpu

ON, OFF = 1, 0


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1807_09932_b200 import binding
    binding.load_library()
    return binding


def kernels_for(eb, B):
    ks = [B.EBIC_KERNEL_DIRECT]
    for k in (B.EBIC_KERNEL_TILED_F32, B.EBIC_KERNEL_RANK8, B.EBIC_KERNEL_PAIRBITS, B.EBIC_KERNEL_UNION_F32,
              B.EBIC_KERNEL_PREFIX, B.EBIC_KERNEL_PAIRTILE):
        try:
            eb.set_kernel(k)
            ks.append(k)
        except B.EbicError:
            pass
    eb.set_kernel(B.EBIC_KERNEL_AUTO)
    return ks


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_counts(eb, B, off, ids, kernel, device=True):
    import torch
    eb.set_kernel(kernel)
    if device:
        c = eb.eval_fitness(dev(off), dev(ids))
        torch.cuda.synchronize()
        out = c.cpu().numpy().view(np.uint64)
    else:
        out = eb.eval_fitness(off, ids)
    eb.set_kernel(B.EBIC_KERNEL_AUTO)
    return out


def gpu_masks(eb, off, ids, chosen, device=True):
    import torch
    ch = np.asarray(chosen, dtype=np.int32)
    if device:
        m, c = eb.extract_rows(dev(off), dev(ids), dev(ch))
        torch.cuda.synchronize()
        return m.cpu().numpy().view(np.uint64), c.cpu().numpy().view(np.uint64)
    return eb.extract_rows(off, ids, ch)


def check_all(B, oracle_mod, matrix, mode, off, ids, chosen=None, expect_status=0):
    """Every kernel's counts and the extraction masks equal the oracle's, element by element."""
    st, want = oracle_mod.eval_fitness(matrix, mode, off, ids)
    assert st == expect_status
    with B.Ebic(matrix, mode) as eb:
        for kern in kernels_for(eb, B):
            for early_exit in ((True, False) if kern != B.EBIC_KERNEL_DIRECT else (True,)):
                eb.set_early_exit(early_exit)
                got = gpu_counts(eb, B, off, ids, kern)
                assert (got == want).all(), (B.KERNEL_NAMES[kern], early_exit, np.flatnonzero(got != want)[:10])
                assert eb.status() == expect_status
        eb.set_early_exit(True)
        n_ind = off.size - 1
        if chosen is None:
            chosen = np.arange(n_ind, dtype=np.int32)
        if len(chosen):
            st, wm, wc = oracle_mod.extract_rows(matrix, mode, off, ids, chosen)
            for use_pairbits in (True, False):                 # pair-table source and float32 source
                eb.set_extract_source(use_pairbits)
                gm, gc = gpu_masks(eb, off, ids, chosen)
                assert (gm == wm).all(), use_pairbits
                assert (gc == wc).all(), use_pairbits
                assert eb.status() == st
    return want


# ------------------------------------------------------------------------- loader (a1, a2, a2')
@pytest.mark.parametrize("rows,cols,nan_rate", [(1, 1, 0.0), (200, 20, 0.1), (513, 33, 0.05), (4097, 100, 0.02)])
def test_loader_products(B, rows, cols, nan_rate):
    rng = np.random.default_rng(rows)
    m = rng.standard_normal((rows, cols), dtype=np.float32)
    m[rng.random((rows, cols)) < nan_rate] = np.nan
    m[0, 0] = np.float32(-0.0) if nan_rate == 0 else m[0, 0]
    if rows >= 200:                                            # values an inexact compare would get wrong
        specials = np.array([0.0, -0.0, np.inf, -np.inf, 1e-45, -1e-45, 1.1754942e-38, 1.1754944e-38, 3.4028235e38,
                             -3.4028235e38, 1.0, np.nextafter(np.float32(1.0), np.float32(2.0))], dtype=np.float32)
        m[5:5 + 64] = rng.choice(specials, size=(64, cols))
        m[70:70 + 32, ::3] = np.nan
    for src in (m, dev(m)):                                    # host pointer and device pointer
        with B.Ebic(src, ON) as eb:
            ld = eb.ld
            assert eb.info(16) == 0                            # no rank tiles while the pair table serves
            eb.set_kernel(B.EBIC_KERNEL_RANK8)                 # builds them on demand
            eb.set_kernel(B.EBIC_KERNEL_AUTO)
            assert ld % 1024 == 0 and ld >= rows and ld - rows < 1024
            mc = eb.debug_read(0)
            assert (mc[:, :rows].view(np.uint32) == m.T.view(np.uint32)).all()   # bit-exact transpose
            assert np.isnan(mc[:, rows:]).all()                                   # padding = missing
            mask = eb.debug_read(1)
            bits = np.unpackbits(mask.view(np.uint8), bitorder="little").reshape(cols, ld).astype(bool)
            assert (bits[:, :rows] == np.isnan(m.T)).all() and bits[:, rows:].all()
            assert (eb.debug_read(2) == (~np.isnan(m)).sum(axis=0).astype(np.uint64)).all()
            rk = eb.debug_read(3)
            below = (m[:, None, :] < m[:, :, None]).sum(axis=2)                   # [rows][cols]
            code = np.where(np.isnan(m), 0x7F, 0x80 | below).astype(np.uint8)
            assert (rk[:, :rows] == code.T).all() and (rk[:, rows:] == 0x7F).all()
            # pair table [a*cols+b][ld/32 words]: bit r = (m[r][b] >= m[r][a]); padding rows 0
            pb = eb.debug_read(4)
            assert eb.info(14) == pb.nbytes
            mp = np.full((ld, cols), np.nan, dtype=np.float32)
            mp[:rows] = m
            with np.errstate(invalid="ignore"):
                ge = mp[:, None, :] >= mp[:, :, None]                              # [ld][a][b]
            want = np.ascontiguousarray(np.packbits(ge.reshape(ld, cols * cols).T, axis=1,
                                                    bitorder="little")).view(np.uint32)
            assert (pb == want).all()
            if cols * cols * 128 + 128 + 4096 <= 232448:       # a 1,024-row tile of all bit columns fits shared memory:
                pbt = eb.debug_read(5)                         # the tile-major copy holds the same words
                assert eb.info(17) == pbt.nbytes
                assert (pbt == want.reshape(cols * cols, ld // 1024, 32).transpose(1, 0, 2)).all()
            else:
                assert eb.info(17) == 0


# ------------------------------------------------------------------------- hand fixtures on the GPU
@pytest.mark.parametrize("name", golden_names())
def test_golden_fixtures_on_gpu(B, oracle_mod, name):
    m, cases = load_golden(name)
    for mode in (ON, OFF):
        sel = [c for c in cases if (c["mode"] == "BOTH" or c["mode"] == ("ON" if mode else "OFF"))]
        off, ids = csr([c["ids"] for c in sel])
        want = check_all(B, oracle_mod, m, mode, off, ids)
        assert want.tolist() == [c["count"] for c in sel]       # and both equal the hand-typed answer
        with B.Ebic(m, mode) as eb:
            gm, gc = gpu_masks(eb, off, ids, np.arange(len(sel)))
            for j, c in enumerate(sel):
                assert (mask_to_bits(gm[j], m.shape[0]) == np.array([ch == "1" for ch in c["mask"]])).all()


# ------------------------------------------------------------------------- the five workloads
@pytest.mark.parametrize("index", [0, 1, 2, 3])
def test_workload_full_size(B, oracle_mod, index):
    w = W.make_workload(index)
    chosen = [k for k, _ in w.planted_individuals][:8] + [w.n_ind - 1]
    check_all(B, oracle_mod, w.matrix, w.missing_mode, w.offsets, w.col_ids, np.array(chosen, np.int32))


def test_workload_c5_scaled(B, oracle_mod):
    """C5's recipe at a size the oracle finishes in seconds: several tiles, a ragged tail (300,001
    rows is not a multiple of 32, 128, 512 or any tile size)."""
    w = W.make_workload(4, rows=300_001, n_ind=512)
    chosen = [k for k, _ in w.planted_individuals][:6]
    check_all(B, oracle_mod, w.matrix, w.missing_mode, w.offsets, w.col_ids, np.array(chosen, np.int32))


@pytest.mark.parametrize("index,rows,n_ind", [(5, None, 1_600), (7, 40_001, 300)])
def test_paper_shaped_workloads(B, oracle_mod, index, rows, n_ind):
    """150 / 310 columns (Table 1 shapes): no rank tiles, at 310 columns no
    float tile of all columns either; every kernel that applies in both early-exit modes, and both extraction
    sources, against the oracle.  P1 at full size, P3 at 40,001 rows (test_paper_shapes_full_size runs P2 and
    P3 at full size)."""
    w = W.make_workload(index, rows=rows, n_ind=n_ind)
    chosen = [k for k, _ in w.planted_individuals][:6] + [w.n_ind - 1]
    check_all(B, oracle_mod, w.matrix, w.missing_mode, w.offsets, w.col_ids, np.array(chosen, np.int32))


def test_planted_recovery_on_gpu(B):
    w = W.make_workload(0)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        chosen = [k for k, _ in w.planted_individuals]
        gm, gc = gpu_masks(eb, w.offsets, w.col_ids, chosen)
        for slot, (k, b) in enumerate(w.planted_individuals):
            assert np.flatnonzero(mask_to_bits(gm[slot], w.rows)).tolist() == w.planted[b].rows.tolist()


# ------------------------------------------------------------------------- edge cases
@pytest.mark.parametrize("rows", [1, 31, 32, 33, 127, 128, 129, 511, 512, 513, 1025, 65_535, 65_536, 65_537])
def test_row_count_edges(B, oracle_mod, rows):
    """Ragged tails around every tile / slab / word size and the paper's old 65,535-row limit."""
    m, off, ids = W.random_case(rows, rows, 7, 40, (0, 7), 0.05, True, False)
    for mode in (ON, OFF):
        check_all(B, oracle_mod, m, mode, off, ids, np.arange(0, 40, 3, dtype=np.int32))


@pytest.mark.parametrize("n_ind", [1, 2, 31, 8191, 8192, 8193, 20_000])
def test_population_size_edges(B, oracle_mod, n_ind):
    """Around the per-launch population chunk (8192) and beyond."""
    m, off, ids = W.random_case(n_ind, 3000, 12, n_ind, (0, 5), 0.03, False, True)
    check_all(B, oracle_mod, m, ON, off, ids, np.array([0, n_ind - 1], np.int32))


def test_population_65536(B, oracle_mod):
    """One more than the paper's population limit of 65,535."""
    m, off, ids = W.random_case(65536, 1000, 10, 65_536, (2, 4), 0.0, False, True)
    check_all(B, oracle_mod, m, OFF, off, ids, np.array([65_535], np.int32))


def test_long_and_degenerate_chromosomes(B, oracle_mod):
    rows, cols = 2000, 16
    m, _, _ = W.random_case(77, rows, cols, 1, (1, 1), 0.02, True, True)
    rng = np.random.default_rng(5)
    inc = np.argsort(m[0])                                         # a long chain some rows can satisfy
    chroms = [[], [3], [3, 3], [3, 3, 3, 3, 3], list(range(cols)), list(range(cols))[::-1],
              inc.tolist(), (inc.tolist() * 3)[:40], rng.integers(0, cols, 1500).tolist(),
              [5] * 1100, rng.integers(0, cols, 33).tolist(), [7, 7, 2, 2]]
    off, ids = csr(chroms)
    for mode in (ON, OFF):
        check_all(B, oracle_mod, m, mode, off, ids)


@pytest.mark.parametrize("rows,cols,n_ind,max_len", [(1, 3, 5, 3), (3_000, 7, 33, 5), (70_001, 40, 1_000, 40),
                                                     (5_003, 32, 300, 80), (200_000, 25, 9_000, 12),
                                                     (160_000, 42, 7_000, 9)])
def test_pairtile_kernel(B, oracle_mod, rows, cols, n_ind, max_len):
    """PAIRTILE (bit-column tiles staged in shared memory, lane = individual): ragged row counts, more tiles than
    SMs and fewer, a population larger than one launch's counters (9,000 at 25 columns: 8,192 + 808; 7,000 at 42
    columns: the tile leaves room for 1,568 counters), chromosomes longer than the 32-entry record, empty / length-1 /
    duplicate-column / invalid individuals, both missing modes, and the
    executed-visit counter (early exit does not apply: executed == nominal)."""
    import torch
    rng = np.random.default_rng(rows + cols)
    m = rng.standard_normal((rows, cols), dtype=np.float32)
    m[rng.random((rows, cols)) < 0.02] = np.nan
    m[: rows // 3] = np.sort(m[: rows // 3], axis=1)           # rows that match increasing-id chromosomes
    chroms = [rng.integers(0, cols, size=rng.integers(0, max_len + 1)).tolist() for _ in range(n_ind)]
    if n_ind > 20:
        chroms[7] = [0, cols]                                  # invalid id: count 0, sticky BAD_COLUMN, others unaffected
        chroms[11] = sorted(rng.permutation(cols)[:min(cols, 6)].tolist())
    off, ids = csr(chroms)
    for mode in (ON, OFF):
        st, want = oracle_mod.eval_fitness(m, mode, off, ids)
        with B.Ebic(m, mode) as eb:
            assert eb.info(17) == eb.info(14) > 0              # the tile-major copy exists: as many bytes as the table
            got = gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_AUTO)
            assert (got == want).all() and eb.last_kernel in (B.EBIC_KERNEL_PAIRTILE, B.EBIC_KERNEL_PAIRBITS)
            if rows < 10_000:                                  # far too small for staged tiles to pay
                assert eb.last_kernel == B.EBIC_KERNEL_PAIRBITS
            eb.status()
            got = gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_PAIRTILE)
            assert (got == want).all(), (mode, np.flatnonzero(got != want)[:10])
            assert eb.last_kernel == B.EBIC_KERNEL_PAIRTILE
            assert eb.status() == st
            eb.set_kernel(B.EBIC_KERNEL_PAIRTILE)
            eb.set_instrumentation(1)
            got = eb.eval_fitness(dev(off), dev(ids))
            torch.cuda.synchronize()
            lens = np.diff(off)
            lens[7 if n_ind > 20 else 0:8 if n_ind > 20 else 0] = 0      # the invalid individual executes nothing
            assert eb.info(10) == eb.ld * int(np.maximum(lens - 1, 0).sum())
            eb.set_instrumentation(0)
            assert (got.cpu().numpy().view(np.uint64) == want).all()
            assert eb.status() == st
            eb.set_tuning(B.TUNE_PT_BUILD, 0)                  # rebuild the table without the tile-major copy
            eb.set_pairbits(False)
            eb.set_pairbits(True)
            assert eb.info(17) == 0 and eb.kernel == B.EBIC_KERNEL_PAIRBITS
            with pytest.raises(B.EbicError):
                eb.set_kernel(B.EBIC_KERNEL_PAIRTILE)


def test_pair_table_beyond_8_gib(B, oracle_mod):
    """A wide matrix whose pair table takes 9.2 GB (150,000 x 700: 490,000 bit columns of 18.8 KB): built by
    ebic_create (cap: 32 GiB and half of the free memory), PAIRBITS and the pair-table extraction against the oracle --
    the 64-bit offsets of a table larger than 2^32 bytes."""
    m, off, ids = W.random_case(700, 150_000, 700, 60, (0, 24), 0.01, False, True)
    st, want = oracle_mod.eval_fitness(m, ON, off, ids)
    chosen = np.array([0, 7, 33, 59], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(m, ON, off, ids, chosen)
    with B.Ebic(m, ON) as eb:
        assert eb.info(14) > 9_000_000_000 and eb.kernel == B.EBIC_KERNEL_PAIRBITS
        for ee in (False, True):
            eb.set_early_exit(ee)
            assert (gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_AUTO) == want).all(), ee
        gm, gc = gpu_masks(eb, off, ids, chosen)
        assert (gm == wm).all() and (gc == wc).all()
        assert eb.status() == st


def test_wide_matrix_falls_back(B, oracle_mod):
    """cols > 127: no rank tiles; cols so large that no float tile of all columns double-buffers: the column-union
    kernel.  The pair table still serves (PAIRBITS); without it AUTO falls back to TILED_F32 / UNION_F32."""
    for cols in (128, 200, 230, 300, 445, 446, 500):
        m, off, ids = W.random_case(cols, 700, cols, 50, (0, 40), 0.02, False, True)
        with B.Ebic(m, ON) as eb:
            with pytest.raises(B.EbicError):
                eb.set_kernel(B.EBIC_KERNEL_RANK8)
            assert eb.kernel == B.EBIC_KERNEL_PAIRBITS
            eb.set_pairbits(False)
            assert eb.info(14) == 0
            expected = B.EBIC_KERNEL_TILED_F32 if cols <= 445 else B.EBIC_KERNEL_UNION_F32
            assert eb.kernel == expected
            with pytest.raises(B.EbicError):
                eb.set_kernel(B.EBIC_KERNEL_PAIRBITS)
            st, want = oracle_mod.eval_fitness(m, ON, off, ids)
            assert (gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_AUTO) == want).all()
            eb.set_pairbits(True)
            assert eb.kernel == B.EBIC_KERNEL_PAIRBITS
        check_all(B, oracle_mod, m, ON, off, ids, np.arange(0, 50, 7, dtype=np.int32))


@pytest.mark.parametrize("cols,batch", [(310, 0), (310, 1), (310, 256), (500, 0), (500, 7), (500, 256), (40, 3), (3000, 0)])
def test_column_union_kernel(B, oracle_mod, cols, batch):
    """SURVEY.md 8(f) NEXT-2 / north_star (3) "(or the population's column union)": with the pair table refused
    (ebic_set_pairbits(0)) a 310- or 500-column matrix runs the column-union kernel, not DIRECT.  Batches of 1
    (every union fits), the default, and 256 individuals (the union overflows the tile: the individuals that do
    not fit are evaluated from global memory by the same warps); chromosomes longer than the 32-id record,
    duplicates and invalid individuals included; both early-exit modes."""
    rows = 2_500
    m, off, ids = W.random_case(cols + batch, rows, cols, 400, (0, 24), 0.02, cols <= 40, True)
    rng = np.random.default_rng(cols)
    extra = [rng.integers(0, cols, 40).tolist(), rng.integers(0, cols, 33).tolist(), [1, 1, 1], [cols - 1, 0],
             rng.permutation(cols)[:min(cols, 300)].tolist(), [0, cols]]           # the last one is invalid
    chroms = [ids[off[k]:off[k + 1]].tolist() for k in range(400)] + extra
    off, ids = csr(chroms)
    st, want = oracle_mod.eval_fitness(m, ON, off, ids)
    assert st == B.EBIC_ERR_BAD_COLUMN
    with B.Ebic(m, ON) as eb:
        eb.set_pairbits(False)
        if cols > 445:                                           # up to 445 columns one 128-row tile of ALL columns still fits
            assert eb.kernel == B.EBIC_KERNEL_UNION_F32          # what AUTO runs now
        elif cols > 127:
            assert eb.kernel == B.EBIC_KERNEL_TILED_F32
        eb.set_kernel(B.EBIC_KERNEL_UNION_F32)
        eb.set_tuning(B.TUNE_UNION_BATCH, batch)
        for early_exit in (True, False):
            eb.set_early_exit(early_exit)
            got = gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_UNION_F32)
            assert (got == want).all(), (early_exit, np.flatnonzero(got != want)[:10])
            assert eb.last_kernel == B.EBIC_KERNEL_UNION_F32
            assert eb.status() == st
        # executed-work accounting: plain work visits every column of every valid chromosome of >= 2 columns
        eb.set_early_exit(False)
        eb.set_instrumentation(1)
        gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_UNION_F32)
        L = np.diff(off)[:-1]
        assert eb.info(10) == eb.ld * int(L[L >= 2].sum())
        eb.set_instrumentation(0)


@pytest.mark.parametrize("sentinel", [999.0, 0.0, -1.5])
def test_sentinel_marks_missing(B, oracle_mod, sentinel):
    """missing cells carry a numeric marker ("e.g. 0 or 999"); ebic_create_sentinel maps it to
    NaN in the loader.  Expected values: the oracle on the matrix with the marker replaced by NaN (input
    preparation by numpy, no method arithmetic).  Cells that already are NaN stay missing; a 0 marker also
    matches -0."""
    m, off, ids = W.random_case(31, 3_001, 40, 120, (0, 8), 0.0, True, True)   # quantised: many 0.0 / -1.5 cells
    rng = np.random.default_rng(5)
    hit = rng.random(m.shape) < 0.03
    m[hit] = np.float32(sentinel)
    m[rng.random(m.shape) < 0.01] = np.float32(np.nan)
    if sentinel == 0.0:
        m[7, 3] = np.float32(-0.0)
    as_nan = m.copy()
    as_nan[m == np.float32(sentinel)] = np.float32(np.nan)
    for mode in (ON, OFF):
        st, want = oracle_mod.eval_fitness(as_nan, mode, off, ids)
        chosen = np.arange(0, 120, 11, dtype=np.int32)
        _, wm, wc = oracle_mod.extract_rows(as_nan, mode, off, ids, chosen)
        for src in (m, dev(m)):                                   # host and device input
            with B.Ebic(src, mode, sentinel=sentinel) as eb:
                assert (eb.debug_read(1) == B.Ebic(as_nan, mode).debug_read(1)).all()      # NaN bitmask
                for kern in kernels_for(eb, B):
                    assert (gpu_counts(eb, B, off, ids, kern) == want).all(), B.KERNEL_NAMES[kern]
                gm, gc = gpu_masks(eb, off, ids, chosen)
                assert (gm == wm).all() and (gc == wc).all()
    with pytest.raises(B.EbicError):
        B.Ebic(m, ON, sentinel=float("nan"))


def test_file_to_counts(B, oracle_mod, tmp_path):
    """The whole ingest side: semicolon-separated file with R-style header (no corner), 999
    as the missing marker -> ebic_read_delimited -> ebic_create_sentinel -> counts and masks equal the oracle's on
    the matrix the file was written from."""
    w = W.make_workload(1, rows=700, n_ind=150)
    marked = w.matrix.copy()
    marked[np.isnan(marked)] = np.float32(999.0)
    lines = [";".join(f"s{c}" for c in range(w.cols))]
    lines += [";".join([f"g{r}"] + [repr(float(v)) for v in marked[r]]) for r in range(w.rows)]
    path = tmp_path / "expr.csv"
    path.write_text("\n".join(lines) + "\n")
    m = B.ebic_read_delimited(path)
    assert m.shape == marked.shape and (m.view(np.uint32) == marked.view(np.uint32)).all()
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    chosen = np.array([k for k, _ in w.planted_individuals][:5], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    with B.Ebic(m, w.missing_mode, sentinel=999.0) as eb:
        assert (gpu_counts(eb, B, w.offsets, w.col_ids, B.EBIC_KERNEL_AUTO) == want).all()
        gm, gc = gpu_masks(eb, w.offsets, w.col_ids, chosen)
        assert (gm == wm).all() and (gc == wc).all()


@pytest.mark.parametrize("knobs", [
    {"TUNE_PB_SMEM_RING": 0},                                    # register-only landing
    {"TUNE_PB_TASKS_PER_SLOT": 2, "TUNE_SORT": 0},               # large chunks, population order
    {"TUNE_PB_TASKS_PER_SLOT": 32, "TUNE_PB_PREFETCH": 0},       # smallest chunks, no L2 prefetch
    {"TUNE_PB_PREFETCH": 3, "TUNE_PDL": 0},                      # distance 3, plain launches
    {"TUNE_PB_PREFETCH": 2, "TUNE_PB_PROLOGUE_CHUNKS": 4},       # the prologue requests more chunks than the distance
    {"TUNE_PDL": 0, "TUNE_SORT": 0, "TUNE_PB_SMEM_RING": 0, "TUNE_PB_PREFETCH": 0},
])
def test_tuning_knobs_keep_parity(B, oracle_mod, knobs):
    """ebic_set_tuning (include/ebic_debug.h) selects other launch configurations / template instantiations of the
    PAIRBITS kernel; each must still reproduce the oracle bit for bit, masks included (the extraction launch is
    chained to the fitness kernel with and without programmatic dependent launch)."""
    import torch
    w = W.make_workload(3, rows=70_001, n_ind=700)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    chosen = np.array([0, 5, 699], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    d_off, d_ids, d_ch = dev(w.offsets), dev(w.col_ids), dev(chosen)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        eb.set_kernel(B.EBIC_KERNEL_PAIRBITS)
        for name, value in knobs.items():
            eb.set_tuning(getattr(B, name), value)
        for ee in (False, True):
            eb.set_early_exit(ee)
            for _ in range(3):                                   # back to back: exercises the launch chaining
                c, m, mc = eb.eval_extract(d_off, d_ids, d_ch)
            torch.cuda.synchronize()
            assert (c.cpu().numpy().view(np.uint64) == want).all(), ee
            assert (m.cpu().numpy().view(np.uint64) == wm).all() and (mc.cpu().numpy().view(np.uint64) == wc).all()
        with pytest.raises(B.EbicError):
            eb.set_tuning(99, 0)
        with pytest.raises(B.EbicError):
            eb.set_tuning(B.TUNE_PB_TASKS_PER_SLOT, 0)


def test_shared_prefix_evaluation(B, oracle_mod):
    """SURVEY.md 8(f) NEXT-4, shared-prefix (trie) evaluation: a CONVERGED population -- 40 parents, every other
    individual a parent with its tail re-drawn -- evaluated by EBIC_KERNEL_PREFIX: counts equal the oracle's, and
    the executed-visit counter shows the shared prefixes were fetched once per group (plain work, early exit off:
    PAIRBITS fetches padded rows * sum(L-1) bit-column rows, PREFIX far fewer); a uniformly random population shares
    almost nothing and must cost no more than the nominal work."""
    import torch
    rows, cols = 30_001, 48
    m, _, _ = W.random_case(77, rows, cols, 1, (1, 1), 0.01, False, True)
    rng = np.random.default_rng(9)
    parents = [rng.permutation(cols)[:rng.integers(8, 21)] for _ in range(40)]
    chroms = []
    for k in range(2_000):
        par = parents[rng.integers(0, len(parents))]
        keep = int(rng.integers(max(2, par.size - 4), par.size + 1))           # shared prefix of keep - 1 pairs
        tail = rng.permutation(cols)[:rng.integers(0, 4)]
        chroms.append(np.concatenate([par[:keep], tail]).tolist())
    chroms += [[], [3], list(range(40)), [5, 5]]                                # L = 0, 1, 40 (never grouped), duplicate
    for name, pop in (("converged", chroms), ("random", None)):
        if pop is None:
            _, off, ids = W.random_case(78, 8, cols, 2_000, (2, 16), 0.0, False, True)
        else:
            off, ids = csr(pop)
        st, want = oracle_mod.eval_fitness(m, ON, off, ids)
        nominal = None
        with B.Ebic(m, ON) as eb:
            nominal = eb.ld * int(np.maximum(np.diff(off) - 1, 0).sum())
            seen = {}
            for kern in (B.EBIC_KERNEL_PAIRBITS, B.EBIC_KERNEL_PREFIX):
                eb.set_kernel(kern)
                for early_exit in (False, True):
                    eb.set_early_exit(early_exit)
                    eb.set_instrumentation(1)
                    got = eb.eval_fitness(dev(off), dev(ids))
                    torch.cuda.synchronize()
                    seen[kern, early_exit] = eb.info(10)
                    eb.set_instrumentation(0)
                    assert (got.cpu().numpy().view(np.uint64) == want).all(), (name, B.KERNEL_NAMES[kern], early_exit)
                    assert eb.last_kernel == kern
            assert seen[B.EBIC_KERNEL_PAIRBITS, False] == nominal
            assert seen[B.EBIC_KERNEL_PREFIX, False] <= nominal
            if name == "converged":
                assert seen[B.EBIC_KERNEL_PREFIX, False] < 0.55 * nominal, seen
            assert eb.status() == 0


def test_ring_path_stress(B, oracle_mod):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.txt), so the PAIRBITS shared-memory landing
    ring is stressed instead: 1,000 evaluations of freshly randomised populations whose chromosomes (9..24 columns)
    all take the ring path, on a matrix of three row chunks with a ragged last step, both early-exit modes, every
    count compared with the oracle.  A write-after-read hazard on the ring would corrupt some AND sooner or later."""
    import torch
    rows, cols, n_ind = 20_001, 24, 192
    m, _, _ = W.random_case(123, rows, cols, 1, (1, 1), 0.01, True, True)
    rng = np.random.default_rng(2024)
    with B.Ebic(m, ON) as eb:
        eb.set_kernel(B.EBIC_KERNEL_PAIRBITS)
        for it in range(1000):
            L = rng.integers(9, cols + 1, n_ind)
            chroms = [rng.permutation(cols)[:l] if it % 3 else rng.integers(0, cols, l) for l in L]
            off, ids = csr(chroms)
            eb.set_early_exit(bool(it & 1))
            got = eb.eval_fitness(dev(off), dev(ids))
            st, want = oracle_mod.eval_fitness(m, ON, off, ids)
            torch.cuda.synchronize()
            got = got.cpu().numpy().view(np.uint64)
            assert (got == want).all(), (it, np.flatnonzero(got != want)[:10])
        assert eb.status() == 0


def test_pairtile_stress(B, oracle_mod):
    """The same stand-in for PAIRTILE's shared-memory paths (tile buffer refilled by TMA behind a barrier, per-lane
    counters, the hand-out cursor of alternating tile parity): 400 evaluations of freshly randomised populations --
    1..700 individuals of 0..40 columns, duplicates allowed every third time -- on a matrix of 40 tiles with a ragged
    last one (fewer tiles than SMs, so most CTAs own a fraction of a tile), every count compared with the oracle."""
    import torch
    rows, cols = 40_500, 24
    m, _, _ = W.random_case(321, rows, cols, 1, (1, 1), 0.01, True, True)
    rng = np.random.default_rng(77)
    with B.Ebic(m, ON) as eb:
        eb.set_kernel(B.EBIC_KERNEL_PAIRTILE)
        for it in range(400):
            n_ind = int(rng.integers(1, 701))
            L = rng.integers(0, 41, n_ind)
            chroms = [rng.permutation(cols)[:min(l, cols)] if it % 3 else rng.integers(0, cols, l) for l in L]
            off, ids = csr(chroms)
            got = eb.eval_fitness(dev(off), dev(ids))
            st, want = oracle_mod.eval_fitness(m, ON, off, ids)
            torch.cuda.synchronize()
            got = got.cpu().numpy().view(np.uint64)
            assert (got == want).all(), (it, n_ind, np.flatnonzero(got != want)[:10])
        assert eb.status() == 0


def test_probe_read_bandwidth(B):
    """Measurement utility: an L2-resident buffer streams faster than HBM; bad arguments are refused."""
    l2 = B.ebic_probe_read_bandwidth(48 << 20, 40)
    hbm = B.ebic_probe_read_bandwidth(2 << 30, 2)
    assert 2_000 < hbm < 9_000 and l2 > hbm
    with pytest.raises(B.EbicError):
        B.ebic_probe_read_bandwidth(1024, 1)
    # the on-chip ceilings of the tiled kernels: 128 B/clk/SM would be ~37 TB/s
    smem = B.ebic_probe_smem_bandwidth()
    fsetp = B.ebic_probe_fsetp_rate()
    assert 10_000 < smem < 60_000, smem
    assert 2_000 < fsetp < 80_000, fsetp
    # PAIRTILE's gather (one slot per lane): conflict-free only with the per-lane rotation of the 16-byte unit
    rotated, plain = B.ebic_probe_smem_gather(True), B.ebic_probe_smem_gather(False)
    assert 10_000 < rotated < 60_000 and plain < rotated / 4, (rotated, plain)


def test_empty_calls(B):
    import torch
    m = np.zeros((10, 3), dtype=np.float32)
    with B.Ebic(m, ON) as eb:
        c = eb.eval_fitness(dev(np.zeros(1, np.int32)), dev(np.zeros(0, np.int32)))
        assert c.numel() == 0
        off, ids = csr([[0, 1]])
        masks, counts = eb.extract_rows(dev(off), dev(ids), torch.zeros(0, dtype=torch.int32, device="cuda"))
        assert masks.shape == (0, 1) and eb.status() == 0


def test_invalid_population_sticky_error(B, oracle_mod):
    m, _, _ = W.random_case(3, 600, 5, 1)
    good = [[0, 1], [2], [], [4, 3, 2]]
    # bad column id
    off, ids = csr(good + [[1, 5], [0, -2, 1]])
    check_all(B, oracle_mod, m, ON, off, ids, expect_status=B.EBIC_ERR_BAD_COLUMN)
    # non-monotone offsets (individual 1), offsets beyond n_ids (last)
    off = np.array([0, 2, 1, 3, 9], dtype=np.int32)
    ids = np.array([0, 1, 2, 3], dtype=np.int32)
    check_all(B, oracle_mod, m, ON, off, ids, expect_status=B.EBIC_ERR_BAD_OFFSETS)
    # offsets that jump BACKWARDS after an invalid individual (round-1 advisor finding): individuals 0, 2 and 3 are
    # valid and overlap in col_ids; nothing the ingest writes may depend on the contents of `offsets`
    off = np.array([0, 10, 5, 8, 12], dtype=np.int32)
    ids = np.array([0, 1, 2, 3, 4, 3, 2, 1, 0, 4, 2, 3], dtype=np.int32)
    check_all(B, oracle_mod, m, ON, off, ids, expect_status=B.EBIC_ERR_BAD_OFFSETS)
    # the same at random: every adjacent pair of random offsets is an individual (half of them invalid), lengths
    # up to 90 ids (beyond the 32-id / 30-pair records), ranges overlapping freely
    rng = np.random.default_rng(11)
    ids = rng.integers(0, 5, 90).astype(np.int32)
    off = rng.integers(0, 91, 301).astype(np.int32)
    for mode in (ON, OFF):
        check_all(B, oracle_mod, m, mode, off, ids, chosen=np.arange(0, 300, 7, dtype=np.int32),
                  expect_status=B.EBIC_ERR_BAD_OFFSETS)
    # chosen index out of range
    off, ids = csr(good)
    with B.Ebic(m, ON) as eb:
        st, wm, wc = oracle_mod.extract_rows(m, ON, off, ids, [1, 9, -1, 0])
        gm, gc = gpu_masks(eb, off, ids, [1, 9, -1, 0])
        assert (gm == wm).all() and (gc == wc).all()
        assert eb.status() == st == B.EBIC_ERR_BAD_OFFSETS
        assert eb.status() == 0                                    # cleared after being read
        # the error does not poison later calls
        assert (gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_AUTO) == oracle_mod.eval_fitness(m, ON, off, ids)[1]).all()


def test_host_pointers_and_streams(B, oracle_mod):
    import torch
    w = W.make_workload(1, rows=5000, n_ind=300)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    chosen = np.array([0, 4, 299], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        # numpy in -> numpy out (host buffers, copies inside the call)
        assert (eb.eval_fitness(w.offsets, w.col_ids) == want).all()
        gm, gc = eb.extract_rows(w.offsets, w.col_ids, chosen)
        assert (gm == wm).all() and (gc == wc).all()
        # pinned host tensors
        po, pi = torch.from_numpy(w.offsets).pin_memory(), torch.from_numpy(w.col_ids).pin_memory()
        out = torch.empty(w.n_ind, dtype=torch.int64).pin_memory()
        eb.eval_fitness(po, pi, counts=out)
        assert (out.numpy().view(np.uint64) == want).all()
        # a non-default stream, stream-ordered with a later copy
        s = torch.cuda.Stream()
        d_off, d_ids = dev(w.offsets), dev(w.col_ids)
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            c = eb.eval_fitness(d_off, d_ids)
            host = c.to("cpu", non_blocking=False)
        assert (host.numpy().view(np.uint64) == want).all()


def test_instrumentation_counts_executed_visits(B):
    w = W.make_workload(4, rows=20_000, n_ind=200)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        nominal = eb.ld * int(w.lengths.sum())
        for kern in (B.EBIC_KERNEL_TILED_F32, B.EBIC_KERNEL_RANK8):
            eb.set_kernel(kern)
            seen = {}
            for early_exit in (False, True):
                eb.set_early_exit(early_exit)
                eb.set_instrumentation(1)
                eb.eval_fitness(dev(w.offsets), dev(w.col_ids))
                seen[early_exit] = eb.info(10)
                eb.set_instrumentation(0)
            assert seen[False] == nominal                          # plain work: executed == nominal
            assert 2 * eb.ld * w.n_ind <= seen[True] <= nominal    # early exit only ever skips columns
        nominal_pairs = eb.ld * int((w.lengths - 1).sum())         # pair kernels count (row, pair) fetches
        for kern in (B.EBIC_KERNEL_PAIRBITS,):
            eb.set_kernel(kern)
            for early_exit in (False, True):
                eb.set_early_exit(early_exit)
                eb.set_instrumentation(1)
                eb.eval_fitness(dev(w.offsets), dev(w.col_ids))
                seen = eb.info(10)
                eb.set_instrumentation(0)
                if early_exit:
                    assert eb.ld * w.n_ind <= seen <= nominal_pairs, B.KERNEL_NAMES[kern]
                else:
                    assert seen == nominal_pairs, B.KERNEL_NAMES[kern]


def test_eval_extract_one_call(B, oracle_mod):
    """ebic_eval_extract = ebic_eval_fitness + ebic_extract_rows on one population: device pointers (extraction
    chained behind the fitness kernel) and host pointers (one upload, one synchronisation); halves skipped when
    n_ind or n_chosen is 0."""
    import torch
    w = W.make_workload(1, rows=9_001, n_ind=500)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    chosen = np.array([0, 3, 499, 7], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        for kern in kernels_for(eb, B):
            eb.set_kernel(kern)
            for use_pairbits in (True, False):
                eb.set_extract_source(use_pairbits)
                c, m, mc = eb.eval_extract(dev(w.offsets), dev(w.col_ids), dev(chosen))
                torch.cuda.synchronize()
                assert (c.cpu().numpy().view(np.uint64) == want).all(), B.KERNEL_NAMES[kern]
                assert (m.cpu().numpy().view(np.uint64) == wm).all() and (mc.cpu().numpy().view(np.uint64) == wc).all()
        eb.set_kernel(B.EBIC_KERNEL_AUTO)
        c, m, mc = eb.eval_extract(w.offsets, w.col_ids, chosen)                 # host buffers
        assert (c == want).all() and (m == wm).all() and (mc == wc).all()
        c, m, mc = eb.eval_extract(w.offsets, w.col_ids, chosen, want_counts=False)
        assert (c == want).all() and (m == wm).all() and mc is None
        c, m, mc = eb.eval_extract(w.offsets, w.col_ids, chosen[:0])             # no extraction
        assert (c == want).all() and m.shape == (0, eb.mask_words)
        assert eb.status() == 0


def test_repeated_calls_replay_a_graph(B, oracle_mod):
    """A GA loop passes the same device buffers every generation: from the second identical call on a non-default
    stream the library captures its launch sequence into a CUDA graph and replays it (include/ebic.h,
    ebic_eval_extract).  Five generations with the population REWRITTEN IN PLACE between them, every kernel, all three
    hot calls: each generation's counts and masks equal the oracle's; a knob change, different buffers, a host-pointer
    call and the default stream all fall back to plain launches."""
    import torch
    rows, cols, n_ind = 70_001, 32, 600
    m, off0, ids0 = W.random_case(321, rows, cols, n_ind, (0, 12), 0.02, False, True)
    side = torch.cuda.Stream()
    chosen = np.array([1, 5, 17, n_ind - 1], dtype=np.int32)
    rng = np.random.default_rng(4)
    with B.Ebic(m, ON) as eb:
        d_off, d_ids, d_ch = dev(off0), dev(ids0), dev(chosen)
        counts = torch.empty(n_ind, dtype=torch.int64, device="cuda")
        masks = torch.empty((len(chosen), eb.mask_words), dtype=torch.int64, device="cuda")
        mcnt = torch.empty(len(chosen), dtype=torch.int64, device="cuda")
        for kern in kernels_for(eb, B):
            eb.set_kernel(kern)
            replayed = 0
            for gen in range(5):
                ids = ids0.copy()
                flip = rng.random(ids.size) < 0.3                      # same CSR shape, new columns
                ids[flip] = rng.integers(0, cols, size=int(flip.sum()), dtype=np.int32)
                d_ids.copy_(torch.from_numpy(ids))
                torch.cuda.synchronize()
                st, want = oracle_mod.eval_fitness(m, ON, off0, ids)
                _, wm, wc = oracle_mod.extract_rows(m, ON, off0, ids, chosen)
                with torch.cuda.stream(side):
                    eb.eval_extract(d_off, d_ids, d_ch, counts=counts, masks=masks, mask_counts=mcnt, stream=side)
                side.synchronize()
                replayed += eb.info(18) > 0
                assert (counts.cpu().numpy().view(np.uint64) == want).all(), (B.KERNEL_NAMES[kern], gen)
                assert (masks.cpu().numpy().view(np.uint64) == wm).all() and (mcnt.cpu().numpy().view(np.uint64) == wc).all()
            assert replayed == 4, (B.KERNEL_NAMES[kern], replayed)     # captured at the second call, held ever since
            n0 = eb.info(8)
            with torch.cuda.stream(side):
                eb.eval_extract(d_off, d_ids, d_ch, counts=counts, masks=masks, mask_counts=mcnt, stream=side)
            side.synchronize()
            assert eb.info(8) - n0 == eb.info(18) >= 2                 # the launch counter follows replays
            # the two single calls are replayed as well
            for _ in range(3):
                with torch.cuda.stream(side):
                    eb.eval_fitness(d_off, d_ids, counts=counts, stream=side)
                side.synchronize()
                assert (counts.cpu().numpy().view(np.uint64) == want).all()
            assert eb.info(18) > 0
            for _ in range(3):
                with torch.cuda.stream(side):
                    eb.extract_rows(d_off, d_ids, d_ch, masks=masks, counts=mcnt, stream=side)
                side.synchronize()
                assert (masks.cpu().numpy().view(np.uint64) == wm).all()
            assert eb.info(18) > 0
            # plain paths: other buffers, the default stream, host pointers, a knob
            other = torch.empty_like(counts)
            with torch.cuda.stream(side):
                eb.eval_fitness(d_off, d_ids, counts=other, stream=side)
            side.synchronize()
            assert eb.info(18) == 0 and (other.cpu().numpy().view(np.uint64) == want).all()
            c = eb.eval_fitness(d_off, d_ids)
            torch.cuda.synchronize()
            assert eb.info(18) == 0 and (c.cpu().numpy().view(np.uint64) == want).all()
            assert (eb.eval_fitness(off0, ids) == want).all()
            eb.set_tuning(B.TUNE_GRAPHS, 0)                            # graphs off
            for _ in range(3):
                with torch.cuda.stream(side):
                    eb.eval_fitness(d_off, d_ids, counts=counts, stream=side)
                side.synchronize()
            assert eb.info(18) == 0 and (counts.cpu().numpy().view(np.uint64) == want).all()
            eb.set_tuning(B.TUNE_GRAPHS, 1)
        assert eb.status() == 0


def test_graph_survives_scratch_reallocation(B, oracle_mod):
    """A captured launch graph holds the addresses of the context's scratch.  A call that cannot be replayed (host
    pointers) with a population four times as large makes the library reallocate that scratch between two replays:
    the graph must be dropped with it, not replayed on freed memory.  Every kernel, against the oracle."""
    import torch
    rows, cols, n_ind = 30_001, 24, 500
    m, off, ids = W.random_case(322, rows, cols, n_ind, (0, 12), 0.02, False, True)
    st, want = oracle_mod.eval_fitness(m, ON, off, ids)
    assert st == 0
    side = torch.cuda.Stream()
    with B.Ebic(m, ON) as eb:
        d_off, d_ids = dev(off), dev(ids)
        counts = torch.empty(n_ind, dtype=torch.int64, device="cuda")
        for i, kern in enumerate(kernels_for(eb, B)):
            eb.set_kernel(kern)                                        # new epoch: the graph logic starts over
            for _ in range(3):
                with torch.cuda.stream(side):
                    eb.eval_fitness(d_off, d_ids, counts=counts, stream=side)
                side.synchronize()
            assert eb.info(18) > 0, B.KERNEL_NAMES[kern]               # a graph is held
            owned = eb.info(9)
            # host pointers and a population twice as large as any before it (the buffers are grown with 25 % headroom,
            # so doubling always outgrows them): scratch regrown
            _, off4, ids4 = W.random_case(323 + i, 1, cols, 2 * n_ind << i, (0, 12))
            st4, want4 = oracle_mod.eval_fitness(m, ON, off4, ids4)
            assert st4 == 0 and (eb.eval_fitness(off4, ids4) == want4).all()
            assert eb.info(9) > owned
            assert eb.info(18) == 0, B.KERNEL_NAMES[kern]              # ... and the graph went with it
            # memory the old scratch occupied may be handed to somebody else: make it so
            junk = [torch.full((1 << 16,), -1, dtype=torch.int64, device="cuda") for _ in range(8)]
            for rep in range(4):
                counts.fill_(-1)
                side.wait_stream(torch.cuda.current_stream())
                with torch.cuda.stream(side):
                    eb.eval_fitness(d_off, d_ids, counts=counts, stream=side)
                side.synchronize()
                assert (counts.cpu().numpy().view(np.uint64) == want).all(), (B.KERNEL_NAMES[kern], rep)
            assert eb.info(18) > 0                                     # captured again on the new buffers
            assert all(bool((j == -1).all()) for j in junk)
        assert eb.status() == 0


def test_extract_into_an_offset_view(B, oracle_mod):
    """include/ebic.h promises uint64 alignment for `masks`, no more: a view that starts 8 bytes into an allocation
    (rows chosen so that a mask is a multiple of 16 bytes long, the case the 16-byte stores serve) must work."""
    import torch
    rows = 128 * 77                                                    # 154 uint64 words per mask: even
    m, off, ids = W.random_case(324, rows, 12, 40, (0, 8), 0.03)
    chosen = np.arange(40, dtype=np.int32)
    st, wm, wc = oracle_mod.extract_rows(m, ON, off, ids, chosen)
    with B.Ebic(m, ON) as eb:
        assert eb.mask_words % 2 == 0
        for use_pairbits in (True, False):
            eb.set_extract_source(use_pairbits)
            for shift in (1, 2, 3):
                buf = torch.zeros(40 * eb.mask_words + shift, dtype=torch.int64, device="cuda")
                masks = buf[shift:].view(40, eb.mask_words)
                assert masks.data_ptr() == buf.data_ptr() + 8 * shift
                gm, gc = eb.extract_rows(dev(off), dev(ids), dev(chosen), masks=masks)
                torch.cuda.synchronize()
                assert (gm.cpu().numpy().view(np.uint64) == wm).all(), (use_pairbits, shift)
                assert (gc.cpu().numpy().view(np.uint64) == wc).all()
                assert (buf[:shift] == 0).all()
        assert eb.status() == st == 0


def test_binding_refuses_wrong_dtypes(B):
    """The C ABI takes raw addresses: the binding must refuse what would be read as garbage (advisor finding)."""
    w = W.make_workload(0)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        with pytest.raises(ValueError, match="int32"):
            eb.eval_fitness(w.offsets.astype(np.int64), w.col_ids)
        with pytest.raises(ValueError, match="int32"):
            eb.eval_fitness(dev(w.offsets), dev(w.col_ids.astype(np.int64)))
        with pytest.raises(ValueError, match="int64"):
            eb.eval_fitness(w.offsets, w.col_ids, counts=np.zeros(w.n_ind, dtype=np.int32))
        with pytest.raises(ValueError, match="mix"):
            eb.eval_fitness(dev(w.offsets), w.col_ids)
        with pytest.raises(ValueError, match="int32"):
            eb.extract_rows(w.offsets, w.col_ids, np.array([0], dtype=np.int64))


# ------------------------------------------------------------------------- row shards on one GPU
@pytest.mark.parametrize("world", [2, 3])
def test_row_shards_through_the_cuda_evaluator(B, oracle_mod, world):
    """The N-GPU path on one GPU, shard by shard: a ragged matrix cut by `row_partition` (64-row seams, which fall
    inside the loader's 1,024-row padding), one ebic context per shard, counts summed and mask shards
    concatenated -- against the UNSHARDED oracle.  What differs from N ranks is only the all-reduce, which the gloo
    tests cover."""
    from paper_1807_09932_b200.sharded import row_partition
    w = W.make_workload(3, rows=5_003, n_ind=300)                # 5,003 = 78 * 64 + 11: ragged last word
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    chosen = np.array([k for k, _ in w.planted_individuals][:4] + [299], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    total = np.zeros(w.n_ind, dtype=np.uint64)
    shards, shard_counts = [], np.zeros(len(chosen), dtype=np.uint64)
    for b, e in row_partition(w.rows, world):
        assert b % 64 == 0
        with B.Ebic(np.ascontiguousarray(w.matrix[b:e]), w.missing_mode) as eb:
            c, m, mc = eb.eval_extract(w.offsets, w.col_ids, chosen)
            total += c
            shards.append(m)
            shard_counts += mc
    assert (total == want).all()
    assert (np.concatenate(shards, axis=1) == wm).all() and (shard_counts == wc).all()


def test_sharded_step_reuses_its_outputs(B, oracle_mod):
    """ShardedEbic.step hands the library the same output tensors every generation, so the captured launch graph is
    replayed from the third generation on whatever the caching allocator does in between; results against the oracle."""
    import torch
    from paper_1807_09932_b200.sharded import ShardedEbic
    w = W.make_workload(3, rows=20_011, n_ind=400)
    chosen = np.array([0, 7, 399], dtype=np.int32)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    _, wm, _ = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    sh = ShardedEbic.from_matrix(w.matrix, w.missing_mode, 0, 1)
    try:
        d_off, d_ids, d_ch = dev(w.offsets), dev(w.col_ids), dev(chosen)
        side = torch.cuda.Stream()
        ptrs = set()
        for gen in range(5):
            churn = [torch.empty(1 << (10 + gen), dtype=torch.int64, device="cuda") for _ in range(4)]   # allocator noise
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                counts, masks = sh.step(d_off, d_ids, d_ch)
            side.synchronize()
            ptrs.add((counts.data_ptr(), masks.data_ptr()))
            assert (counts.cpu().numpy().view(np.uint64) == want).all(), gen
            assert (masks.cpu().numpy().view(np.uint64) == wm).all(), gen
            if gen >= 2:
                assert sh.ebic.info(18) > 0, gen                   # replayed
            del churn
        assert len(ptrs) == 1
        assert sh.ebic.status(side) == 0
    finally:
        sh.close()


def test_bench_two_ranks_on_one_device(oracle_mod):
    """The N > 1 branch of bench.py (row shards, ShardedEbic.step, the all-reduce, the rank-0 line) as two gloo ranks
    that share this one GPU: exit code 0, one JSON line, and the fingerprint of the all-reduced counts equals the
    oracle's counts on the unsharded matrix.  Timings of such a run mean nothing and are not looked at."""
    import hashlib
    import json
    import os
    import socket
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(root / "bench.py"), "--gpus", "2", "--dist-backend", "gloo", "--one-device",
           "--workload", "c3", "--steps", "2", "--warmup", "3", "--no-per-workload", "--no-cpu-baseline"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root, env=dict(os.environ))
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, res.stdout[-2000:]
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "strong" and "functional_check_only" in out["config"]
    w = W.make_workload(2)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    assert st == 0
    assert out["counts_sha256_16"] == hashlib.sha256(want.astype(np.uint64).tobytes()).hexdigest()[:16]


# ------------------------------------------------------------------------- full sizes against the oracle
@pytest.mark.parametrize("index", [6, 7])
def test_paper_shapes_full_size(B, oracle_mod, index):
    """P2 (54,675 x 178, 1,600 individuals) and P3 (436,444 x 310, 1,600 individuals) at FULL size: every count of
    the kernel AUTO picks and of the float32 kernels that apply, and the masks of 9 individuals from both
    extraction sources, word for word against the oracle."""
    import torch
    w = W.make_workload(index)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    chosen = np.array([k for k, _ in w.planted_individuals][:8] + [w.n_ind - 1], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    d_off, d_ids = dev(w.offsets), dev(w.col_ids)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        assert eb.kernel == B.EBIC_KERNEL_PAIRBITS
        for kern in kernels_for(eb, B):
            eb.set_kernel(kern)
            got = eb.eval_fitness(d_off, d_ids)
            torch.cuda.synchronize()
            assert (got.cpu().numpy().view(np.uint64) == want).all(), B.KERNEL_NAMES[kern]
        eb.set_kernel(B.EBIC_KERNEL_AUTO)
        for use_pairbits in (True, False):
            eb.set_extract_source(use_pairbits)
            gm, gc = gpu_masks(eb, w.offsets, w.col_ids, chosen)
            assert (gm == wm).all() and (gc == wc).all(), use_pairbits
        assert eb.status() == 0


def test_c5_full_size(B, oracle_mod):
    """BASELINE.json configs[4] at FULL size (16,777,216 rows x 32 columns, 4,096 individuals), in the launch
    configuration bench.py times: the oracle evaluates ALL 4,096 individuals (about 5.5e11 comparisons, 1-2
    minutes on the box's host cores) and every GPU kernel's counts are compared with it element by element; the
    masks of 8 planted individuals from both extraction sources are compared with oracle.extract_rows word for
    word (BASELINE.json north_star: "bit-exact fitness counts and row bitmasks vs the oracle on all five configs")."""
    import torch
    w = W.make_workload(4)
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    assert st == 0
    chosen = np.array([k for k, _ in w.planted_individuals][:8], dtype=np.int32)
    _, wm, wc = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    assert (wc == want[chosen]).all()
    d_off, d_ids = dev(w.offsets), dev(w.col_ids)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        eb.set_early_exit(False)                                 # bench.py's headline configuration
        got = eb.eval_fitness(d_off, d_ids)
        torch.cuda.synchronize()
        assert eb.last_kernel == B.EBIC_KERNEL_PAIRTILE          # what AUTO (and bench.py) runs on C5
        assert (got.cpu().numpy().view(np.uint64) == want).all()
        for kern in (B.EBIC_KERNEL_PAIRTILE, B.EBIC_KERNEL_PAIRBITS, B.EBIC_KERNEL_RANK8, B.EBIC_KERNEL_TILED_F32,
                     B.EBIC_KERNEL_DIRECT):
            eb.set_kernel(kern)
            for early_exit in ((True,) if kern == B.EBIC_KERNEL_DIRECT else (True, False)):
                eb.set_early_exit(early_exit)
                c = eb.eval_fitness(d_off, d_ids)
                torch.cuda.synchronize()
                got = c.cpu().numpy().view(np.uint64)
                assert (got == want).all(), (B.KERNEL_NAMES[kern], early_exit, np.flatnonzero(got != want)[:10])
        eb.set_kernel(B.EBIC_KERNEL_AUTO)
        for use_pairbits in (True, False):
            eb.set_extract_source(use_pairbits)
            gm, gc = gpu_masks(eb, w.offsets, w.col_ids, chosen)
            assert (gm == wm).all() and (gc == wc).all(), use_pairbits
        # the fused call, as bench.py's step issues it
        c, m, mc = eb.eval_extract(d_off, d_ids, dev(chosen))
        torch.cuda.synchronize()
        assert (c.cpu().numpy().view(np.uint64) == want).all() and (m.cpu().numpy().view(np.uint64) == wm).all()
        for slot, (k, b) in enumerate(w.planted_individuals[:8]):
            assert mask_to_bits(wm[slot], w.rows)[w.planted[b].clean_rows].all()      # planted rows are matched
        assert eb.status() == 0
