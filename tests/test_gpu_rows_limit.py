"""The paper's headline capability -- "up to 2^31-1 rows per single GPU" ("Support for Big Data") --
through the C ABI against the oracle: one matrix with exactly 2^31-1 rows (2 columns, 17.2 GB) and one of more than
2^31 ELEMENTS with real width (70,000,001 x 32, ragged: not a multiple of 64).  Every product c * ld + r, r * cols,
(ld / 32) * n_ind, every grid dimension and every 16-byte-unit offset of the pair table crosses 2^31 (or 2^32 bytes)
here.  Bit-exact, like the rest of the suite.

The tests need about 45 GB of host memory and 45 GB of HBM; they skip (loudly) on a box that has less.
"""
from __future__ import annotations

import numpy as np
import pytest

from conftest import csr
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


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host_bytes_available() -> int:
    import psutil
    avail = psutil.virtual_memory().available
    try:                                                       # a container's own limit, when it has one
        limit = open("/sys/fs/cgroup/memory.max").read().strip()
        used = int(open("/sys/fs/cgroup/memory.current").read())
        if limit != "max":
            avail = min(avail, int(limit) - used)
    except OSError:
        pass
    return avail


def need(host_gb: float, device_gb: float):
    import torch
    if host_bytes_available() < host_gb * 2**30:
        pytest.skip(f"needs {host_gb} GB of host memory, {host_bytes_available() / 2**30:.0f} GB available")
    if torch.cuda.mem_get_info()[0] < device_gb * 2**30:
        pytest.skip(f"needs {device_gb} GB of device memory")


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


def check_against_oracle(B, oracle_mod, m, mode, off, ids, chosen, expect_kernels):
    import torch
    rows = m.shape[0]
    st, want = oracle_mod.eval_fitness(m, mode, off, ids)
    st2, wm, wc = oracle_mod.extract_rows(m, mode, off, ids, chosen)
    assert st == 0 and st2 == 0 and (wc == want[chosen]).all()
    d_off, d_ids, d_ch = dev(off), dev(ids), dev(chosen)
    with B.Ebic(m, mode) as eb:
        assert eb.ld % 1024 == 0 and 0 <= eb.ld - rows < 1024 and eb.mask_words == (rows + 63) // 64
        ks = kernels_for(eb, B)
        assert set(expect_kernels) <= set(ks), [B.KERNEL_NAMES[k] for k in ks]
        for kern in ks:
            eb.set_kernel(kern)
            for early_exit in ((True, False) if kern != B.EBIC_KERNEL_DIRECT else (True,)):
                eb.set_early_exit(early_exit)
                got = eb.eval_fitness(d_off, d_ids)
                torch.cuda.synchronize()
                got = got.cpu().numpy().view(np.uint64)
                assert (got == want).all(), (B.KERNEL_NAMES[kern], early_exit, got, want)
        eb.set_kernel(B.EBIC_KERNEL_AUTO)
        eb.set_early_exit(True)
        for use_pairbits in (True, False):                     # pair-table source and float32 source
            eb.set_extract_source(use_pairbits)
            gm, gc = eb.extract_rows(d_off, d_ids, d_ch)
            torch.cuda.synchronize()
            gc = gc.cpu().numpy().view(np.uint64)
            gm = gm.cpu().numpy().view(np.uint64)
            assert (gc == wc).all(), use_pairbits
            assert (gm == wm).all(), use_pairbits
            assert (np.bitwise_count(gm).sum(axis=1, dtype=np.uint64) == gc).all()     # popcount == count
            if rows % 64:
                assert not (gm[:, -1] >> np.uint64(rows % 64)).any()                   # bits >= rows are zero
            del gm
        # the host-pointer route of the same call (staging + copy back of 2^25-word masks)
        got = eb.eval_fitness(off, ids)
        assert (got == want).all()
        assert eb.status() == 0


@pytest.mark.parametrize("mode", [ON, OFF])
def test_rows_2_pow_31_minus_1(B, oracle_mod, mode):
    """rows = 2^31 - 1, the largest row count ebic_create accepts, 2 columns: Mc is 17.2 GB, one mask
    2^25 words with exactly one dead bit at the top.  NaN in the first and last row, around 2^24 (float32's integer
    limit) and at 2^30, plus a few thousand at random."""
    need(45, 45)
    rows = 2**31 - 1
    nan_rows = [0, 1, 2**24 - 1, 2**24, 2**24 + 1, 2**30, 2**30 + 1, rows - 2, rows - 1, rows - 1]
    m = W.big_matrix(1, rows, 2, levels=4, n_nan=3000, nan_rows=nan_rows)
    assert np.isnan(m[rows - 1]).all()
    off, ids = csr([[], [0], [1], [0, 1], [1, 0], [0, 1, 0], [0, 0]])
    chosen = np.arange(7, dtype=np.int32)
    check_against_oracle(B, oracle_mod, m, mode, off, ids, chosen,
                         [B.EBIC_KERNEL_PAIRTILE, B.EBIC_KERNEL_PAIRBITS, B.EBIC_KERNEL_RANK8, B.EBIC_KERNEL_TILED_F32])


def test_more_than_2_pow_31_elements(B, oracle_mod):
    """70,000,001 x 32 = 2.24e9 elements (9 GB; ld * cols * 4 > 2^33 bytes; 68,360 PAIRTILE tiles; pair table
    1,024 bit columns of 8.75 MB = 9 GB), 64 individuals of 0 .. 40 columns (repeats allowed, so chromosomes run past
    the 30-pair records and the 32-id records), missing values on."""
    need(45, 45)
    rows, cols = 70_000_001, 32
    m = W.big_matrix(2, rows, cols, levels=3, n_nan=50_000, nan_rows=[0, rows - 1, 2**26, 2**26 + 1])
    rng = np.random.default_rng(77)
    chrom = [rng.integers(0, cols, size=int(L)).astype(np.int32) for L in rng.integers(0, 41, size=60)]
    chrom += [np.arange(32, dtype=np.int32), np.arange(31, -1, -1, dtype=np.int32), np.array([5], dtype=np.int32),
              np.array([], dtype=np.int32)]
    off, ids = csr(chrom)
    chosen = np.array([0, 13, 60, 61, 62, 63], dtype=np.int32)
    check_against_oracle(B, oracle_mod, m, ON, off, ids, chosen,
                         [B.EBIC_KERNEL_PAIRTILE, B.EBIC_KERNEL_PAIRBITS, B.EBIC_KERNEL_RANK8, B.EBIC_KERNEL_TILED_F32])
