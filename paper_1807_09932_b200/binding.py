"""Thin Python binding over libebic.so (the C ABI of include/ebic.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library.  PyTorch is used for device
memory and streams only.  If the library is missing or no CUDA device is present the calls raise
-- there is no CPU fallback.

Module-level functions carry the C names (`ebic_create`, `ebic_eval_fitness`, ...) and take raw
pointers / sizes.  `Ebic` is the convenience wrapper the tests and bench.py use: it accepts torch
CUDA tensors (device pointers) or numpy arrays / CPU tensors (host pointers) and passes their
addresses straight through.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional

import numpy as np

EBIC_OK = 0
EBIC_ERR_ARG = 1
EBIC_ERR_OOM = 2
EBIC_ERR_CUDA = 3
EBIC_ERR_BAD_COLUMN = 4
EBIC_ERR_BAD_OFFSETS = 5
EBIC_ERR_IO = 6
EBIC_ERR_LIMIT = 7
EBIC_NOALLOC_MAX_IND = 16384
EBIC_MISSING_OFF = 0
EBIC_MISSING_ON = 1
EBIC_KERNEL_AUTO = 0
EBIC_KERNEL_DIRECT = 1
EBIC_KERNEL_TILED_F32 = 2
EBIC_KERNEL_RANK8 = 3
EBIC_KERNEL_PAIRBITS = 4
EBIC_KERNEL_UNION_F32 = 5
EBIC_KERNEL_PREFIX = 6
EBIC_KERNEL_PAIRTILE = 7
KERNEL_NAMES = {0: "auto", 1: "direct", 2: "tiled_f32", 3: "rank8", 4: "pairbits", 5: "union_f32", 6: "prefix",
                7: "pairtile"}
# ebic_set_tuning knobs (include/ebic_debug.h)
(TUNE_PB_TASKS_PER_SLOT, TUNE_PB_PREFETCH, TUNE_PB_SMEM_RING, TUNE_SORT, TUNE_PDL, TUNE_UNION_BATCH, TUNE_PT_BUILD,
 TUNE_PT_MIN_WORK, TUNE_PB_PROLOGUE_CHUNKS, TUNE_GRAPHS, TUNE_PB_INGEST_PREFETCH) = range(11)

LIB_PATH = Path(__file__).resolve().parent / "libebic.so"

# every symbol include/ebic.h (the boundary) declares: (restype, argtypes)
_vp, _i32, _i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
_f64p = ctypes.POINTER(ctypes.c_double)
SYMBOLS = {
    "ebic_create": (ctypes.c_int, [_vp, _i64, _i32, _i32, ctypes.POINTER(_vp)]),
    "ebic_create_sentinel": (ctypes.c_int, [_vp, _i64, _i32, _i32, ctypes.c_float, ctypes.POINTER(_vp)]),
    "ebic_destroy": (ctypes.c_int, [_vp]),
    "ebic_eval_fitness": (ctypes.c_int, [_vp, _vp, _vp, _i32, _i64, _vp, _vp]),
    "ebic_eval_fitness_noalloc": (ctypes.c_int, [_vp, _vp, _vp, _i32, _i64, _vp, _vp]),
    "ebic_extract_rows": (ctypes.c_int, [_vp, _vp, _vp, _i32, _i64, _vp, _i32, _vp, _vp, _vp]),
    "ebic_eval_extract": (ctypes.c_int, [_vp, _vp, _vp, _i32, _i64, _vp, _vp, _i32, _vp, _vp, _vp]),
    "ebic_mask_words": (_i64, [_vp]),
    "ebic_status": (ctypes.c_int, [_vp, _vp]),
    "ebic_read_delimited": (ctypes.c_int, [ctypes.c_char_p, ctypes.c_char, ctypes.POINTER(ctypes.POINTER(ctypes.c_float)),
                                           ctypes.POINTER(_i64), ctypes.POINTER(_i32)]),
    "ebic_free_host": (None, [_vp]),
    "ebic_strerror": (ctypes.c_char_p, [ctypes.c_int]),
}
# every symbol include/ebic_debug.h declares (knobs, read-backs, probes for tests and bench.py)
DEBUG_SYMBOLS = {
    "ebic_set_kernel": (ctypes.c_int, [_vp, _i32]),
    "ebic_set_pairbits": (ctypes.c_int, [_vp, _i32]),
    "ebic_set_extract_source": (ctypes.c_int, [_vp, _i32]),
    "ebic_set_early_exit": (ctypes.c_int, [_vp, _i32]),
    "ebic_set_tuning": (ctypes.c_int, [_vp, _i32, _i32]),
    "ebic_set_instrumentation": (ctypes.c_int, [_vp, _i32]),
    "ebic_get_info": (_i64, [_vp, _i32]),
    "ebic_debug_read": (ctypes.c_int, [_vp, _i32, _vp, _i64]),
    "ebic_probe_read_bandwidth": (ctypes.c_int, [_i64, _i32, _f64p]),
    "ebic_probe_smem_bandwidth": (ctypes.c_int, [_f64p]),
    "ebic_probe_smem_gather": (ctypes.c_int, [_i32, _f64p]),
    "ebic_probe_fsetp_rate": (ctypes.c_int, [_f64p]),
}

_lib = None


class EbicError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: status {status} ({strerror(status)})")


def load_library() -> ctypes.CDLL:
    """Load libebic.so; raises (loudly) when it has not been built."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1807_09932_b200.csrc.build` "
                "(there is no CPU fallback)")
        lib = ctypes.CDLL(str(LIB_PATH))
        for name, (res, args) in {**SYMBOLS, **DEBUG_SYMBOLS}.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def strerror(status: int) -> str:
    try:
        return load_library().ebic_strerror(int(status)).decode()
    except Exception:
        return "?"


# ---------------------------------------------------------------- C names, raw pointers
def ebic_create(matrix_ptr: int, rows: int, cols: int, missing_mode: int) -> int:
    out = _vp()
    st = load_library().ebic_create(matrix_ptr, rows, cols, missing_mode, ctypes.byref(out))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_create")
    return out.value


def ebic_create_sentinel(matrix_ptr: int, rows: int, cols: int, missing_mode: int, sentinel: float) -> int:
    out = _vp()
    st = load_library().ebic_create_sentinel(matrix_ptr, rows, cols, missing_mode, float(sentinel), ctypes.byref(out))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_create_sentinel")
    return out.value


def ebic_destroy(ctx: int) -> None:
    load_library().ebic_destroy(ctx)


def ebic_eval_fitness(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, counts_ptr, stream=0) -> None:
    st = load_library().ebic_eval_fitness(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, counts_ptr, stream)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_eval_fitness")


def ebic_eval_fitness_noalloc(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, counts_ptr, stream=0) -> None:
    st = load_library().ebic_eval_fitness_noalloc(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, counts_ptr, stream)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_eval_fitness_noalloc")


def ebic_extract_rows(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, chosen_ptr, n_chosen, masks_ptr,
                      counts_ptr, stream=0) -> None:
    st = load_library().ebic_extract_rows(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, chosen_ptr, n_chosen,
                                          masks_ptr, counts_ptr, stream)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_extract_rows")


def ebic_eval_extract(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, counts_ptr, chosen_ptr, n_chosen, masks_ptr,
                      mask_counts_ptr, stream=0) -> None:
    st = load_library().ebic_eval_extract(ctx, offsets_ptr, col_ids_ptr, n_ind, n_ids, counts_ptr, chosen_ptr, n_chosen,
                                          masks_ptr, mask_counts_ptr, stream)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_eval_extract")


def ebic_mask_words(ctx) -> int:
    return int(load_library().ebic_mask_words(ctx))


def ebic_status(ctx, stream=0) -> int:
    return int(load_library().ebic_status(ctx, stream))


def ebic_set_kernel(ctx, kernel: int) -> None:
    st = load_library().ebic_set_kernel(ctx, kernel)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_set_kernel")


def ebic_set_pairbits(ctx, on: bool) -> None:
    st = load_library().ebic_set_pairbits(ctx, 1 if on else 0)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_set_pairbits")


def ebic_set_extract_source(ctx, use_pairbits: bool) -> None:
    load_library().ebic_set_extract_source(ctx, 1 if use_pairbits else 0)


def ebic_set_early_exit(ctx, on: bool) -> None:
    load_library().ebic_set_early_exit(ctx, 1 if on else 0)


def ebic_set_tuning(ctx, knob: int, value: int) -> None:
    st = load_library().ebic_set_tuning(ctx, int(knob), int(value))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_set_tuning")


def ebic_set_instrumentation(ctx, on: int) -> None:
    load_library().ebic_set_instrumentation(ctx, int(on))


def ebic_get_info(ctx, what: int) -> int:
    return int(load_library().ebic_get_info(ctx, what))


def ebic_debug_read(ctx, what: int, dst: np.ndarray) -> None:
    st = load_library().ebic_debug_read(ctx, what, dst.ctypes.data, dst.nbytes)
    if st != EBIC_OK:
        raise EbicError(st, "ebic_debug_read")


def ebic_read_delimited(path: str, delimiter: str = "") -> np.ndarray:
    """ebic_read_delimited: float32 [rows][cols] copied out of the library's buffer (which is then freed)."""
    lib = load_library()
    m = ctypes.POINTER(ctypes.c_float)()
    rows, cols = _i64(0), _i32(0)
    d = delimiter.encode() if delimiter else b"\0"
    st = lib.ebic_read_delimited(str(path).encode(), d, ctypes.byref(m), ctypes.byref(rows), ctypes.byref(cols))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_read_delimited")
    try:
        return np.ctypeslib.as_array(m, shape=(rows.value, cols.value)).copy()
    finally:
        lib.ebic_free_host(ctypes.cast(m, _vp))


# ---------------------------------------------------------------- convenience wrapper
def ebic_probe_read_bandwidth(buffer_bytes: int, reps: int) -> float:
    out = ctypes.c_double(0.0)
    st = load_library().ebic_probe_read_bandwidth(int(buffer_bytes), int(reps), ctypes.byref(out))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_probe_read_bandwidth")
    return out.value


def ebic_probe_smem_bandwidth() -> float:
    out = ctypes.c_double(0.0)
    st = load_library().ebic_probe_smem_bandwidth(ctypes.byref(out))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_probe_smem_bandwidth")
    return out.value


def ebic_probe_smem_gather(rotate: bool = True) -> float:
    out = ctypes.c_double(0.0)
    st = load_library().ebic_probe_smem_gather(1 if rotate else 0, ctypes.byref(out))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_probe_smem_gather")
    return out.value


def ebic_probe_fsetp_rate() -> float:
    out = ctypes.c_double(0.0)
    st = load_library().ebic_probe_fsetp_rate(ctypes.byref(out))
    if st != EBIC_OK:
        raise EbicError(st, "ebic_probe_fsetp_rate")
    return out.value


def _require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("ebic-b200 needs a CUDA device (B200, sm_100a); there is no CPU fallback")
    return torch


def _ptr(a) -> int:
    """Address of a torch tensor (CPU or CUDA) or numpy array; the array must be contiguous."""
    if a is None:
        return 0
    if isinstance(a, np.ndarray):
        if not a.flags.c_contiguous:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    if not a.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return a.data_ptr()


def _is_cuda(a) -> bool:
    return (not isinstance(a, np.ndarray)) and a.is_cuda


def _itemsize_kind(a):
    """(itemsize, kind) of a numpy array or torch tensor; kind 'i' / 'u' / 'f' / '?'."""
    if isinstance(a, np.ndarray):
        return a.dtype.itemsize, a.dtype.kind
    name = str(a.dtype)
    kind = "f" if ("float" in name or "bfloat" in name) else "u" if "uint" in name else "i" if "int" in name else "?"
    return a.element_size(), kind


def _check_args(where: str, device_index: int, int32_args, int64_args):
    """The C ABI takes raw addresses, so a wrong dtype or device would be read as garbage: refuse it here.
    int32_args: offsets / col_ids / chosen (int32); int64_args: counts / masks (int64 or uint64).  All arguments
    must be of one kind (all CUDA tensors on the context's device, or all host arrays)."""
    kinds = set()
    for name, a in list(int32_args.items()) + list(int64_args.items()):
        if a is None:
            continue
        size, kind = _itemsize_kind(a)
        want = 4 if name in int32_args else 8
        if kind not in ("i", "u") or size != want or (want == 4 and kind != "i"):
            raise ValueError(f"{where}: `{name}` must be {'int32' if want == 4 else 'int64 / uint64'}, got {a.dtype}")
        if _is_cuda(a):
            if a.device.index != device_index:
                raise ValueError(f"{where}: `{name}` is on cuda:{a.device.index}, the context on cuda:{device_index}")
            kinds.add("cuda")
        else:
            kinds.add("host")
    if len(kinds) > 1:
        raise ValueError(f"{where}: arguments must be all CUDA tensors or all host arrays, not a mix")


def _stream_handle(stream) -> int:
    torch = _require_cuda()
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class Ebic:
    """One loaded matrix (ebic_ctx).  matrix: float32 [rows][cols], torch CUDA/CPU tensor or numpy."""

    def __init__(self, matrix, missing_mode: int, sentinel: Optional[float] = None):
        """`sentinel`: numeric value that marks missing cells in `matrix` (ebic_create_sentinel); None = NaN only."""
        torch = _require_cuda()
        load_library()
        if isinstance(matrix, np.ndarray):
            if matrix.dtype != np.float32 or matrix.ndim != 2:
                raise ValueError("matrix must be float32 [rows][cols]")
            matrix = np.ascontiguousarray(matrix)
        else:
            if matrix.dtype != torch.float32 or matrix.dim() != 2:
                raise ValueError("matrix must be float32 [rows][cols]")
            matrix = matrix.contiguous()
            if matrix.is_cuda:
                torch.cuda.current_stream().synchronize()      # ebic_create runs on the legacy stream
        self.rows, self.cols = int(matrix.shape[0]), int(matrix.shape[1])
        self.missing_mode = int(missing_mode)
        self.device_index = int(torch.cuda.current_device())
        if _is_cuda(matrix) and matrix.device.index != self.device_index:
            raise ValueError(f"matrix is on cuda:{matrix.device.index}, the current device is cuda:{self.device_index}")
        if sentinel is None:
            self._ctx = ebic_create(_ptr(matrix), self.rows, self.cols, self.missing_mode)
        else:
            self._ctx = ebic_create_sentinel(_ptr(matrix), self.rows, self.cols, self.missing_mode, sentinel)
        self.mask_words = ebic_mask_words(self._ctx)

    # -- lifetime
    def close(self):
        if getattr(self, "_ctx", None):
            ebic_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the two hot calls
    def eval_fitness(self, offsets, col_ids, counts=None, stream=None):
        """counts (uint64 bit pattern in an int64 tensor / uint64 numpy array) for the whole population.

        Device tensors in -> device tensor out, asynchronous on `stream` (default: torch's current
        stream).  numpy / CPU tensors in -> numpy uint64 out, synchronous (host buffers, the copies
        happen inside the call).
        """
        torch = _require_cuda()
        _check_args("eval_fitness", self.device_index, {"offsets": offsets, "col_ids": col_ids}, {"counts": counts})
        n_ind = int(offsets.shape[0]) - 1
        n_ids = int(col_ids.shape[0])
        if _is_cuda(offsets):
            if counts is None:
                counts = torch.empty(n_ind, dtype=torch.int64, device=offsets.device)
        elif counts is None:
            counts = np.empty(n_ind, dtype=np.uint64)
        ebic_eval_fitness(self._ctx, _ptr(offsets), _ptr(col_ids), n_ind, n_ids, _ptr(counts),
                          _stream_handle(stream))
        return counts

    def eval_fitness_noalloc(self, offsets, col_ids, counts, stream=None):
        """ebic_eval_fitness_noalloc: the same counts as eval_fitness, from a call that allocates no device memory.

        For GA loops inside a host that has handed the rest of the HBM to its own pool, or that must not stall the
        device with cudaFree / cudaMalloc once it is running (see include/ebic.h).  All three arguments are CUDA
        tensors the caller made during set-up -- `counts` (int64 [n_ind]) included, the wrapper allocates nothing
        either.  At most EBIC_NOALLOC_MAX_IND individuals (EbicError with status EBIC_ERR_LIMIT beyond that); every
        call on a GPU shares one fixed scratch array, so keep such calls on one stream.  Returns `counts`.
        """
        if counts is None or not (_is_cuda(offsets) and _is_cuda(col_ids) and _is_cuda(counts)):
            raise ValueError("eval_fitness_noalloc: offsets, col_ids and counts must be CUDA tensors supplied by the caller")
        _check_args("eval_fitness_noalloc", self.device_index, {"offsets": offsets, "col_ids": col_ids}, {"counts": counts})
        n_ind = int(offsets.shape[0]) - 1
        if int(counts.shape[0]) < n_ind:
            raise ValueError("eval_fitness_noalloc: `counts` is shorter than the population")
        ebic_eval_fitness_noalloc(self._ctx, _ptr(offsets), _ptr(col_ids), n_ind, int(col_ids.shape[0]), _ptr(counts),
                                  _stream_handle(stream))
        return counts

    def extract_rows(self, offsets, col_ids, chosen, masks=None, counts=None, want_counts=True, stream=None):
        """(masks [n_chosen][mask_words], counts [n_chosen] or None) for the chosen individuals."""
        masks, counts = self._extract_outputs("extract_rows", offsets, col_ids, chosen, masks, counts, want_counts)
        ebic_extract_rows(self._ctx, _ptr(offsets), _ptr(col_ids), int(offsets.shape[0]) - 1, int(col_ids.shape[0]),
                          _ptr(chosen), int(chosen.shape[0]), _ptr(masks), _ptr(counts), _stream_handle(stream))
        return masks, counts

    def _extract_outputs(self, where, offsets, col_ids, chosen, masks, counts, want_counts):
        torch = _require_cuda()
        _check_args(where, self.device_index, {"offsets": offsets, "col_ids": col_ids, "chosen": chosen},
                    {"masks": masks, "mask_counts": counts})
        n_chosen = int(chosen.shape[0])
        if _is_cuda(offsets):
            if masks is None:
                masks = torch.empty((n_chosen, self.mask_words), dtype=torch.int64, device=offsets.device)
            if counts is None and want_counts:
                counts = torch.empty(n_chosen, dtype=torch.int64, device=offsets.device)
        else:
            if masks is None:
                masks = np.empty((n_chosen, self.mask_words), dtype=np.uint64)
            if counts is None and want_counts:
                counts = np.empty(n_chosen, dtype=np.uint64)
        return masks, counts

    def eval_extract(self, offsets, col_ids, chosen, counts=None, masks=None, mask_counts=None, want_counts=True,
                     stream=None):
        """ebic_eval_extract: one GA generation -> (counts [n_ind], masks [n_chosen][mask_words], mask_counts)."""
        torch = _require_cuda()
        _check_args("eval_extract", self.device_index, {"offsets": offsets, "col_ids": col_ids}, {"counts": counts})
        n_ind = int(offsets.shape[0]) - 1
        if counts is None:
            counts = (torch.empty(n_ind, dtype=torch.int64, device=offsets.device) if _is_cuda(offsets)
                      else np.empty(n_ind, dtype=np.uint64))
        masks, mask_counts = self._extract_outputs("eval_extract", offsets, col_ids, chosen, masks, mask_counts, want_counts)
        ebic_eval_extract(self._ctx, _ptr(offsets), _ptr(col_ids), n_ind, int(col_ids.shape[0]), _ptr(counts),
                          _ptr(chosen), int(chosen.shape[0]), _ptr(masks), _ptr(mask_counts), _stream_handle(stream))
        return counts, masks, mask_counts

    # -- status / knobs / introspection
    def status(self, stream=None) -> int:
        return ebic_status(self._ctx, _stream_handle(stream))

    def set_kernel(self, kernel: int) -> None:
        ebic_set_kernel(self._ctx, kernel)

    def set_pairbits(self, on: bool) -> None:
        ebic_set_pairbits(self._ctx, on)

    def set_extract_source(self, use_pairbits: bool) -> None:
        ebic_set_extract_source(self._ctx, use_pairbits)

    def set_early_exit(self, on: bool) -> None:
        ebic_set_early_exit(self._ctx, on)

    def set_instrumentation(self, on: int) -> None:
        ebic_set_instrumentation(self._ctx, on)

    def set_tuning(self, knob: int, value: int) -> None:
        ebic_set_tuning(self._ctx, knob, value)

    def create_breakdown_ms(self) -> dict:
        """ebic_create's time by phase (CUDA events inside the library)."""
        names = ["h2d_transpose_pad", "nan_mask", "pair_table", "rank_tiles", "total"]
        return {n: self.info(20 + i) / 1e6 for i, n in enumerate(names)}

    def info(self, what: int) -> int:
        return ebic_get_info(self._ctx, what)

    @property
    def ld(self) -> int:
        return self.info(2)

    @property
    def kernel(self) -> int:
        return self.info(4)

    @property
    def last_kernel(self) -> int:
        """Kernel of the last fitness launch 0 = none yet."""
        return self.info(15)

    def debug_read(self, what: int) -> np.ndarray:
        ld, cols = self.ld, self.cols
        if what == 0:
            dst = np.empty((cols, ld), dtype=np.float32)
        elif what == 1:
            dst = np.empty((cols, ld // 32), dtype=np.uint32)
        elif what == 2:
            dst = np.empty(cols, dtype=np.uint64)
        elif what == 3:
            dst = np.empty((cols, ld), dtype=np.uint8)
        elif what == 4:
            dst = np.empty((cols * cols, ld // 32), dtype=np.uint32)
        elif what == 5:
            dst = np.empty((ld // 1024, cols * cols, 32), dtype=np.uint32)
        else:
            raise ValueError(what)
        ebic_debug_read(self._ctx, what, dst)
        return dst
