"""ebic_eval_fitness_noalloc against the existing path (ebic_eval_fitness) and the oracle.

Why the call exists: ebic_eval_fitness grows its per-call scratch with cudaFree + cudaMalloc whenever a population
is larger than any before it.  A GA loop embedded in a service that gave the rest of the HBM to its own pool at
start-up, or that runs beside latency-bound streams a device-wide cudaFree would stall, cannot afford that in the
middle of a run.  The no-allocation call keeps the same records in one fixed 2,176 KiB array inside libebic.so
(at most EBIC_NOALLOC_MAX_IND = 16,384 individuals), shared by every call on the GPU.

What is checked: counts bit-exact (tolerance 0, as everywhere in this suite) against ebic_eval_fitness and the
oracle on consecutive calls -- the array still holds the previous, differently sized population each time --,
including two calls queued on one stream with no synchronisation between them; the limit and the host-pointer
refusals; and that free device memory does not move across calls.

The file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
Nothing in it depends on what ran before (own contexts, own tensors; the array needs no particular contents).
"""
from __future__ import annotations

import numpy as np
import pytest

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


def populations(cols, sizes, seed):
    rng = np.random.default_rng([7, seed])
    # lengths 0..40: empty and single-column individuals, and chromosomes past the 30 pairs a record holds
    return [W.make_population(rng, cols, n, (0, 40)) for n in sizes]


def existing_path(eb, off, ids):
    import torch
    c = eb.eval_fitness(dev(off), dev(ids))
    torch.cuda.synchronize()
    return c.cpu().numpy().view(np.uint64)


@pytest.mark.parametrize("pair_table", [True, False])
@pytest.mark.parametrize("mode", [ON, OFF])
def test_consecutive_calls_match_the_existing_path(B, oracle_mod, pair_table, mode):
    """Calls in a row, each on a population of another size than the one before: the fixed array is full of the
    previous call's records every time.  PAIRBITS (pair table) and DIRECT (no pair table) variants."""
    import torch
    m, _, _ = W.random_case(31, 5000 if pair_table else 3000, 48, 1, nan_rate=0.03, ties=True)
    pops = populations(48, [700, 300, 1500, 64, 65], seed=mode)
    with B.Ebic(m, mode) as eb:
        if not pair_table:
            eb.set_pairbits(False)
        for early_exit in (True, False):
            eb.set_early_exit(early_exit)
            for off, ids in pops:
                want = existing_path(eb, off, ids)
                st, ref = oracle_mod.eval_fitness(m, mode, off, ids)
                assert st == 0 and (want == ref).all()
                out = torch.full((off.size - 1,), -1, dtype=torch.int64, device="cuda")
                got = eb.eval_fitness_noalloc(dev(off), dev(ids), out)
                torch.cuda.synchronize()
                got = got.cpu().numpy().view(np.uint64)
                assert (got == want).all(), (pair_table, mode, early_exit, off.size - 1, np.flatnonzero(got != want)[:10])
                assert eb.status() == 0


def test_two_calls_queued_back_to_back(B, oracle_mod):
    """Two calls on one stream, nothing between them: the second call's ingest must wait for the first call's
    fitness kernel, which is still reading the shared array."""
    import torch
    m, _, _ = W.random_case(32, 40000, 24, 1, nan_rate=0.02)
    (off1, ids1), (off2, ids2) = populations(24, [2000, 900], seed=3)
    with B.Ebic(m, ON) as eb:
        want1, want2 = existing_path(eb, off1, ids1), existing_path(eb, off2, ids2)
        assert (want1 == oracle_mod.eval_fitness(m, ON, off1, ids1)[1]).all()
        assert (want2 == oracle_mod.eval_fitness(m, ON, off2, ids2)[1]).all()
        d = [dev(a) for a in (off1, ids1, off2, ids2)]
        out1 = torch.empty(2000, dtype=torch.int64, device="cuda")
        out2 = torch.empty(900, dtype=torch.int64, device="cuda")
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        for _ in range(3):
            out1.fill_(-1), out2.fill_(-1)
            stream.wait_stream(torch.cuda.current_stream())
            eb.eval_fitness_noalloc(d[0], d[1], out1, stream=stream)
            eb.eval_fitness_noalloc(d[2], d[3], out2, stream=stream)
            stream.synchronize()
            assert (out1.cpu().numpy().view(np.uint64) == want1).all()
            assert (out2.cpu().numpy().view(np.uint64) == want2).all()
        assert eb.status(stream) == 0


def test_invalid_individuals_and_sticky_status(B, oracle_mod):
    """Validation is the existing path's: a bad individual gets 0, its neighbours are unaffected, the status sticks."""
    import torch
    m, off, ids = W.random_case(33, 2000, 16, 200, len_range=(2, 9))
    ids = ids.copy()
    ids[off[17]] = 16                                           # column id outside [0, cols)
    st, ref = oracle_mod.eval_fitness(m, OFF, off, ids)
    assert st == B.EBIC_ERR_BAD_COLUMN and ref[17] == 0
    with B.Ebic(m, OFF) as eb:
        want = existing_path(eb, off, ids)
        assert eb.status() == B.EBIC_ERR_BAD_COLUMN
        out = torch.empty(200, dtype=torch.int64, device="cuda")
        got = eb.eval_fitness_noalloc(dev(off), dev(ids), out)
        assert eb.status() == B.EBIC_ERR_BAD_COLUMN             # synchronises the stream
        assert (got.cpu().numpy().view(np.uint64) == want).all() and (want == ref).all()
        assert eb.status() == 0


def test_limit_and_refusals(B, oracle_mod):
    """The largest population the array holds works; one more is refused with EBIC_ERR_LIMIT before anything runs;
    host buffers are refused (they would need a staging allocation)."""
    import torch
    n_max = B.EBIC_NOALLOC_MAX_IND
    m, _, _ = W.random_case(34, 1500, 12, 1, nan_rate=0.05)
    rng = np.random.default_rng(34)
    off, ids = W.make_population(rng, 12, n_max + 1, (0, 5))
    with B.Ebic(m, ON) as eb:
        d_off, d_ids = dev(off), dev(ids)
        out = torch.full((n_max + 1,), -7, dtype=torch.int64, device="cuda")
        with pytest.raises(B.EbicError) as exc:
            eb.eval_fitness_noalloc(d_off, d_ids, out)
        assert exc.value.status == B.EBIC_ERR_LIMIT and "EBIC_NOALLOC_MAX_IND" in str(exc.value)
        torch.cuda.synchronize()
        assert (out == -7).all()                                # nothing was launched
        # exactly the maximum: the first n_max individuals of the same CSR
        off_max = off[:n_max + 1]
        n_ids = int(off_max[-1])
        want = existing_path(eb, off_max, ids[:n_ids])
        assert (want == oracle_mod.eval_fitness(m, ON, off_max, ids[:n_ids])[1]).all()
        got = eb.eval_fitness_noalloc(dev(off_max), dev(ids[:n_ids]), out[:n_max])
        torch.cuda.synchronize()
        assert (got.cpu().numpy().view(np.uint64) == want).all()
        # host pointers: the wrapper refuses, and so does the C entry point itself
        with pytest.raises(ValueError):
            eb.eval_fitness_noalloc(off_max, ids[:n_ids], np.empty(n_max, dtype=np.uint64))
        h_out = np.empty(n_max, dtype=np.uint64)
        st = B.load_library().ebic_eval_fitness_noalloc(eb._ctx, off_max.ctypes.data, ids.ctypes.data, n_max, n_ids,
                                                        h_out.ctypes.data, None)
        assert st == B.EBIC_ERR_ARG
        assert eb.status() == 0


def test_free_device_memory_does_not_move(B):
    """Growing populations make ebic_eval_fitness reallocate; the no-allocation call must leave cudaMemGetInfo's
    free figure where it was.  Every tensor is made, and every kernel variant run once, before the measurement."""
    import torch
    m, _, _ = W.random_case(35, 20000, 20, 1)
    pops = populations(20, [100, 400, 1600, 6400, 16384], seed=5)
    with B.Ebic(m, ON) as eb:
        d = [(dev(off), dev(ids), torch.empty(off.size - 1, dtype=torch.int64, device="cuda")) for off, ids in pops]
        eb.eval_fitness_noalloc(*d[0])                          # set-up call: address look-up, lazy kernel loading
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        owned0 = eb.info(9)
        for args in d:
            eb.eval_fitness_noalloc(*args)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
        assert eb.info(9) == owned0                             # the context's own buffers did not grow either
        assert eb.status() == 0
