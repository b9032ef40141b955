"""Row-sharded multi-GPU evaluation ("full multi-GPU
support", rows are what is split over GPUs).

One process per GPU (`torch.distributed`).  Rows are cut into contiguous slices whose lengths are
multiples of 64 (so a 64-bit mask word never straddles two ranks); every rank holds all columns of
its slice and the whole (small) population.  The path has exactly ONE exchange step: the per-rank
counts are summed with an all-reduce of int64[n_ind] (NCCL over NVLink on GPUs; 12.8-32 KB, so it
is latency-bound -- which is why small inputs do not scale, consistent with the paper's 1.2x at
12k rows against 6.6x at 436k rows on 8 GPUs).  Row bitmasks stay sharded: rank
i owns words [row_begin/64, row_end/64); `gather_masks` concatenates them with one all-gather when a
caller wants them whole.

`ShardedEbic.from_matrix` is the product path: it loads the rank's row slice into a `binding.Ebic`
context on the current CUDA device, and the counts never leave the device before the all-reduce.
The constructor with injected evaluators exists so that the host logic (partition, reduce, gather)
can be tested on CPU with gloo.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Tuple

import numpy as np


def row_partition(rows: int, world_size: int) -> List[Tuple[int, int]]:
    """Contiguous [begin, end) row slices, one per rank; every boundary except the last is a multiple
    of 64; slices differ by at most 64 rows; ranks beyond the data get empty slices."""
    if rows <= 0 or world_size <= 0:
        raise ValueError("rows and world_size must be positive")
    words = (rows + 63) // 64
    base, extra = divmod(words, world_size)
    bounds, w = [], 0
    for r in range(world_size):
        n = base + (1 if r < extra else 0)
        b, e = min(rows, w * 64), min(rows, (w + n) * 64)
        bounds.append((b, e))
        w += n
    return bounds


class ShardedEbic:
    """Fitness evaluation over a row-sharded matrix.

    local_eval(offsets, col_ids) -> int64 counts of THIS rank's row slice (torch tensor on the
    reduce device, or numpy).  local_extract(offsets, col_ids, chosen) -> uint64/int64 masks
    [n_chosen][local_words] of this rank's slice.  `device`: where a rank with an EMPTY slice puts its
    zero counts / empty masks (NCCL needs CUDA tensors on every rank); None = CPU (gloo).
    """

    def __init__(self, rows: int, rank: int, world_size: int, local_eval: Callable,
                 local_extract: Optional[Callable] = None, group=None, device=None):
        self.rows, self.rank, self.world_size = int(rows), int(rank), int(world_size)
        self.bounds = row_partition(self.rows, self.world_size)
        self.row_begin, self.row_end = self.bounds[self.rank]
        self._eval, self._extract, self._group = local_eval, local_extract, group
        self.device = device
        self.ebic = None

    @classmethod
    def from_matrix(cls, matrix, missing_mode: int, rank: int, world_size: int, group=None,
                    rows_total: Optional[int] = None, sentinel: Optional[float] = None):
        """The CUDA path.  `matrix`: the WHOLE float32 [rows][cols] matrix (numpy / torch; the rank's slice
        is cut here), or -- with `rows_total` given -- only this rank's slice [row_begin, row_end) of a
        matrix of `rows_total` rows.  The slice is loaded into a `binding.Ebic` context on the current CUDA
        device; a rank whose slice is empty gets no context."""
        import torch
        from . import binding
        device = torch.device("cuda", torch.cuda.current_device())
        rows = int(matrix.shape[0]) if rows_total is None else int(rows_total)
        self = cls(rows, rank, world_size, None, None, group=group, device=device)
        local = matrix[self.row_begin:self.row_end] if rows_total is None else matrix
        if int(local.shape[0]) != self.local_rows:
            raise ValueError(f"rank {rank}: slice has {int(local.shape[0])} rows, the partition gives {self.local_rows}")
        if self.local_rows > 0:
            self.ebic = binding.Ebic(local, missing_mode, sentinel=sentinel)
            self._eval = self.ebic.eval_fitness
            self._extract = lambda off, ids, ch: self.ebic.extract_rows(off, ids, ch, want_counts=False)[0]
        return self

    def close(self):
        if self.ebic is not None:
            self.ebic.close()
            self.ebic = None

    @property
    def local_rows(self) -> int:
        return self.row_end - self.row_begin

    @property
    def local_words(self) -> int:
        return (self.local_rows + 63) // 64

    def _zeros(self, shape):
        import torch
        return torch.zeros(shape, dtype=torch.int64, device=self.device if self.device is not None else "cpu")

    def eval_fitness(self, offsets, col_ids):
        """Whole-matrix counts on every rank: local counts, then one all-reduce(SUM)."""
        import torch
        import torch.distributed as dist
        n_ind = int(offsets.shape[0]) - 1
        if self.local_rows > 0:
            local = self._eval(offsets, col_ids)
            if isinstance(local, np.ndarray):
                local = torch.from_numpy(local.astype(np.int64, copy=False))
                if self.device is not None:
                    local = local.to(self.device)
        else:
            local = self._zeros(n_ind)
        if self.world_size > 1:
            dist.all_reduce(local, op=dist.ReduceOp.SUM, group=self._group)
        return local

    def extract_rows(self, offsets, col_ids, chosen):
        """This rank's shard of the masks: words [row_begin/64, ceil(row_end/64))."""
        if self.local_rows == 0:
            return self._zeros((int(chosen.shape[0]), 0))
        return self._extract(offsets, col_ids, chosen)

    def step(self, offsets, col_ids, chosen):
        """One generation: (whole-matrix counts on every rank, this rank's mask shard).  On the CUDA path the
        local half is one `ebic_eval_extract` call into tensors that are reused every generation (copy what must
        outlive the next `step`)."""
        import torch.distributed as dist
        if self.ebic is None:
            return self.eval_fitness(offsets, col_ids), self.extract_rows(offsets, col_ids, chosen)
        counts, masks = self._step_buffers(int(offsets.shape[0]) - 1, int(chosen.shape[0]), offsets)
        self.ebic.eval_extract(offsets, col_ids, chosen, counts=counts, masks=masks, want_counts=False)
        if self.world_size > 1:
            dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=self._group)
        return counts, masks

    def _step_buffers(self, n_ind: int, n_chosen: int, like):
        """The output tensors `step` hands to the library and to the all-reduce, made once per (population size,
        number chosen) and reused every generation: with the same pointers in every call the library's captured
        launch graph stays valid (include/ebic.h, ebic_eval_extract) instead of depending on the caching allocator
        returning the same addresses.  The tensors `step` returns are therefore overwritten by the next `step`."""
        import torch
        if not getattr(like, "is_cuda", False):                    # host arrays: the binding makes numpy outputs
            return None, None
        key = (n_ind, n_chosen)
        if getattr(self, "_step_key", None) != key:
            self._step_out = (torch.empty(n_ind, dtype=torch.int64, device=like.device),
                              torch.empty((n_chosen, self.ebic.mask_words), dtype=torch.int64, device=like.device))
            self._step_key = key
        return self._step_out

    def gather_masks(self, local_masks):
        """Concatenate every rank's mask shard along the word axis (all ranks get the whole mask): ONE
        all-gather of shards padded to the widest one (shards differ by at most one word)."""
        import torch
        import torch.distributed as dist
        if isinstance(local_masks, np.ndarray):
            local_masks = torch.from_numpy(local_masks.view(np.int64).copy())
            if self.device is not None:
                local_masks = local_masks.to(self.device)
        if self.world_size == 1:
            return local_masks
        words = [(e - b + 63) // 64 for b, e in self.bounds]
        n_chosen, widest = int(local_masks.shape[0]), max(words)
        mine = torch.zeros((n_chosen, widest), dtype=local_masks.dtype, device=local_masks.device)
        mine[:, :words[self.rank]] = local_masks
        everyone = torch.empty((self.world_size, n_chosen, widest), dtype=mine.dtype, device=mine.device)
        dist.all_gather(list(everyone.unbind(0)), mine, group=self._group)     # one collective, preallocated output
        return torch.cat([everyone[r, :, :words[r]] for r in range(self.world_size)], dim=1)
