"""Parity of the CUDA path (through the C ABI, via the thin binding) against the CPU oracle.

Bar: bit-exact (integer counts and bitmasks from exact float32 comparisons; tolerance 0).
Every fitness kernel (DIRECT, TILED_F32, RANK8, PAIRBITS) is compared with the oracle on the same seeded
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
    for k in (B.EBIC_KERNEL_TILED_F32, B.EBIC_KERNEL_RANK8, B.EBIC_KERNEL_PAIRBITS):
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
    for src in (m, dev(m)):                                    # host pointer and device pointer
        with B.Ebic(src, ON) as eb:
            ld = eb.ld
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


@pytest.mark.parametrize("index,rows,n_ind", [(5, None, 1_600), (6, None, 400), (7, 40_001, 300)])
def test_paper_shaped_workloads(B, oracle_mod, index, rows, n_ind):
    """150 / 178 / 310 columns (Table 1 shapes): no rank tiles, at 310 columns
    no float tile either; every kernel that applies, and both extraction sources, against the oracle.  P1 at
    full size; P2 with a quarter of the population and P3 at 40,001 rows to keep the oracle to seconds."""
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


def test_wide_matrix_falls_back(B, oracle_mod):
    """cols > 127: no rank tiles; cols so large that no float tile double-buffers: DIRECT only.  The pair
    table still serves (PAIRBITS); without it AUTO falls back to TILED_F32 / DIRECT."""
    for cols in (128, 200, 500):
        m, off, ids = W.random_case(cols, 700, cols, 50, (0, 9), 0.02, False, True)
        with B.Ebic(m, ON) as eb:
            with pytest.raises(B.EbicError):
                eb.set_kernel(B.EBIC_KERNEL_RANK8)
            assert eb.kernel == B.EBIC_KERNEL_PAIRBITS
            eb.set_pairbits(False)
            assert eb.info(14) == 0
            expected = B.EBIC_KERNEL_TILED_F32 if cols <= 200 else B.EBIC_KERNEL_DIRECT
            assert eb.kernel == expected
            with pytest.raises(B.EbicError):
                eb.set_kernel(B.EBIC_KERNEL_PAIRBITS)
            st, want = oracle_mod.eval_fitness(m, ON, off, ids)
            assert (gpu_counts(eb, B, off, ids, B.EBIC_KERNEL_AUTO) == want).all()
            eb.set_pairbits(True)
            assert eb.kernel == B.EBIC_KERNEL_PAIRBITS
        check_all(B, oracle_mod, m, ON, off, ids, np.arange(0, 50, 7, dtype=np.int32))


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


@pytest.mark.parametrize("env", [
    {"EBIC_PB_SMEM": "0"},                                       # register-only landing
    {"EBIC_PB_WARPS": "8", "EBIC_PB_TASKS_PER_SLOT": "2"},       # 8-warp CTAs, large chunks
    {"EBIC_PB_WARPS": "1", "EBIC_PB_PREFETCH": "0"},             # 1-warp CTAs, no L2 prefetch
    {"EBIC_PB_WARM": "3", "EBIC_PB_PREFETCH": "2"},              # warm prefetch from ingest, distance 2
    {"EBIC_PB_PERSIST": "1"},                                    # persistent warps drawing tasks from a counter
])
def test_experiment_knobs_keep_parity(env):
    """The PAIRBITS experiment knobs (environment variables read once per process) select other
    template instantiations of the kernel; each must still reproduce the oracle bit for bit.  Runs in a child
    process because the knobs are latched at first use."""
    import os
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    code = (
        "import numpy as np, torch, oracle\n"
        "from paper_1807_09932_b200 import binding as B, workloads as W\n"
        "w = W.make_workload(3, rows=70_001, n_ind=700)\n"
        "st, want = oracle.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)\n"
        "with B.Ebic(w.matrix, w.missing_mode) as eb:\n"
        "    eb.set_kernel(B.EBIC_KERNEL_PAIRBITS)\n"
        "    for ee in (False, True):\n"
        "        eb.set_early_exit(ee)\n"
        "        got = eb.eval_fitness(torch.from_numpy(w.offsets).cuda(), torch.from_numpy(w.col_ids).cuda())\n"
        "        torch.cuda.synchronize()\n"
        "        assert (got.cpu().numpy().view(np.uint64) == want).all(), ee\n"
        "print('ok')\n")
    res = subprocess.run([sys.executable, "-c", code], cwd=root, env={**os.environ, **env}, capture_output=True,
                         text=True, timeout=600)
    assert res.returncode == 0 and res.stdout.strip().endswith("ok"), res.stderr[-2000:]


def test_probe_read_bandwidth(B):
    """Measurement utility: an L2-resident buffer streams faster than HBM; bad arguments are refused."""
    l2 = B.ebic_probe_read_bandwidth(64 << 20, 20)
    hbm = B.ebic_probe_read_bandwidth(2 << 30, 2)
    assert 2_000 < hbm < 9_000 and l2 > hbm
    with pytest.raises(B.EbicError):
        B.ebic_probe_read_bandwidth(1024, 1)


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


# ------------------------------------------------------------------------- full-size C5 (bench config)
def test_c5_full_size_sampled(B, oracle_mod):
    """BASELINE.json configs[4] at full size, in the launch configuration bench.py times: a sample of
    individuals against the oracle one by one, plus properties that hold at any size."""
    w = W.make_workload(4)
    d_off, d_ids = dev(w.offsets), dev(w.col_ids)
    rng = np.random.default_rng(99)
    sample = np.unique(np.concatenate([[k for k, _ in w.planted_individuals][:16],
                                       rng.choice(w.n_ind, 32, replace=False)])).astype(np.int32)
    sub_off, sub_ids = csr([w.col_ids[w.offsets[k]:w.offsets[k + 1]].tolist() for k in sample])
    st, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, sub_off, sub_ids)
    with B.Ebic(w.matrix, w.missing_mode) as eb:
        import torch
        results = {}
        eb.eval_fitness(d_off, d_ids)
        assert eb.last_kernel == B.EBIC_KERNEL_PAIRBITS          # what AUTO (and bench.py --workload c5) runs
        for kern in (B.EBIC_KERNEL_RANK8, B.EBIC_KERNEL_TILED_F32, B.EBIC_KERNEL_PAIRBITS):
            eb.set_kernel(kern)
            for early_exit in (False, True):
                eb.set_early_exit(early_exit)
                c = eb.eval_fitness(d_off, d_ids)
                torch.cuda.synchronize()
                results[kern] = c.cpu().numpy().view(np.uint64)
                assert (results[kern][sample] == want).all(), (B.KERNEL_NAMES[kern], early_exit)
        for kern in results:
            assert (results[kern] == results[B.EBIC_KERNEL_RANK8]).all(), B.KERNEL_NAMES[kern]
        counts = results[B.EBIC_KERNEL_RANK8]
        # properties: planted rows are a subset; popcount(mask) == count; tail bits zero
        chosen = np.array([k for k, _ in w.planted_individuals][:4], dtype=np.int32)
        gm, gc = gpu_masks(eb, w.offsets, w.col_ids, chosen)
        for slot, (k, b) in enumerate(w.planted_individuals[:4]):
            bits = mask_to_bits(gm[slot], w.rows)
            assert bits[w.planted[b].clean_rows].all()
            assert int(bits.sum()) == int(gc[slot]) == int(counts[k])
        # closed form on uniformly random individuals: count ~ Binomial(rows, (1-p)^L / L!) on the rows
        # that are iid; planted rows (sorted in some column order) can shift it either way, by at most
        # the number of planted rows in biclusters sharing a column with the individual.
        import math
        p = w.cfg.nan_rate
        first_random = 4 * len(w.planted)
        for k in range(first_random, first_random + 200):
            L = int(w.lengths[k])
            if L > 5:
                continue
            chrom = set(w.col_ids[w.offsets[k]:w.offsets[k + 1]].tolist())
            affected = sum(b.rows.size for b in w.planted if chrom & set(b.order.tolist()))
            q = (1 - p) ** L / math.factorial(L)
            sigma = math.sqrt(w.rows * q * (1 - q))
            assert abs(int(counts[k]) - w.rows * q) <= 6 * sigma + affected, (k, L, int(counts[k]), w.rows * q)
        # third witness on the whole population: the simple DIRECT kernel
        eb.set_kernel(B.EBIC_KERNEL_DIRECT)
        c = eb.eval_fitness(d_off, d_ids)
        torch.cuda.synchronize()
        assert (c.cpu().numpy().view(np.uint64) == counts).all()
