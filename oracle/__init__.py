"""CPU oracle for the EBIC fitness / row-extraction path.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with the CUDA path in
``paper_1807_09932_b200`` and neither imports the other.

The arithmetic lives in ``ebic_oracle.c`` (plain C, see its header for the definition, the
PAPER.md passages and the readings it follows).  This file only compiles that C file with gcc
(``-O2``, never ``-ffast-math``) and marshals numpy arrays into it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ebic_oracle.c"
_LIB = _HERE / "libebic_oracle.so"

OK = 0
ERR_ARG = 1
ERR_BAD_COLUMN = 4
ERR_BAD_OFFSETS = 5
MISSING_OFF = 0
MISSING_ON = 1

_lib = None


def build(force: bool = False) -> Path:
    """Compile ebic_oracle.c -> libebic_oracle.so next to it (gcc -O2 -fopenmp, no fast-math)."""
    if not force and _LIB.exists() and _LIB.stat().st_mtime >= _SRC.stat().st_mtime:
        return _LIB
    tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
           "-fno-fast-math", "-o", str(tmp), str(_SRC)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(str(build()))
        f32p = ctypes.POINTER(ctypes.c_float)
        i32p = ctypes.POINTER(ctypes.c_int32)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        lib.oracle_eval_fitness.restype = ctypes.c_int
        lib.oracle_eval_fitness.argtypes = [f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32,
                                            i32p, i32p, ctypes.c_int32, ctypes.c_int64, u64p,
                                            ctypes.c_int32]
        lib.oracle_extract_rows.restype = ctypes.c_int
        lib.oracle_extract_rows.argtypes = [f32p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int32,
                                            i32p, i32p, ctypes.c_int32, ctypes.c_int64, i32p,
                                            ctypes.c_int32, u64p, u64p]
        lib.oracle_max_threads.restype = ctypes.c_int
        lib.oracle_max_threads.argtypes = []
        _lib = lib
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if a.ndim != 2:
        raise ValueError("matrix must be 2-D [rows][cols]")
    return a


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32).reshape(-1)


def _ptr(a, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def eval_fitness(matrix, missing_mode, offsets, col_ids, n_threads: int = 0):
    """-> (status, counts uint64[n_ind]).  matrix: float32 row-major [rows][cols]."""
    lib = _load()
    m = _f32(matrix)
    off = _i32(offsets)
    ids = _i32(col_ids)
    n_ind = off.size - 1
    if n_ind < 0:
        raise ValueError("offsets must have n_ind+1 entries")
    counts = np.zeros(max(n_ind, 0), dtype=np.uint64)
    ids_buf = ids if ids.size else np.zeros(1, dtype=np.int32)
    st = lib.oracle_eval_fitness(_ptr(m, ctypes.c_float), m.shape[0], m.shape[1], int(missing_mode),
                                 _ptr(off, ctypes.c_int32), _ptr(ids_buf, ctypes.c_int32), n_ind,
                                 ids.size, _ptr(counts, ctypes.c_uint64), int(n_threads))
    return int(st), counts


def extract_rows(matrix, missing_mode, offsets, col_ids, chosen):
    """-> (status, masks uint64[n_chosen][ceil(rows/64)], counts uint64[n_chosen])."""
    lib = _load()
    m = _f32(matrix)
    off = _i32(offsets)
    ids = _i32(col_ids)
    ch = _i32(chosen)
    n_ind = off.size - 1
    words = (m.shape[0] + 63) // 64
    masks = np.zeros((ch.size, words), dtype=np.uint64)
    counts = np.zeros(ch.size, dtype=np.uint64)
    ids_buf = ids if ids.size else np.zeros(1, dtype=np.int32)
    ch_buf = ch if ch.size else np.zeros(1, dtype=np.int32)
    st = lib.oracle_extract_rows(_ptr(m, ctypes.c_float), m.shape[0], m.shape[1], int(missing_mode),
                                 _ptr(off, ctypes.c_int32), _ptr(ids_buf, ctypes.c_int32), n_ind,
                                 ids.size, _ptr(ch_buf, ctypes.c_int32), ch.size,
                                 _ptr(masks, ctypes.c_uint64), _ptr(counts, ctypes.c_uint64))
    return int(st), masks, counts
