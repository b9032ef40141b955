"""Shared test helpers.  GPU tests carry @pytest.mark.gpu; everything else runs on CPU."""
from __future__ import annotations

import math
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

GOLDEN = Path(__file__).resolve().parent / "golden"


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def load_golden(name: str):
    """Parse a tests/golden/*.txt fixture -> (matrix float32, [case dict])."""
    rows = cols = None
    matrix, cases = [], []
    in_matrix = False
    for raw in (GOLDEN / name).read_text().splitlines():
        line = raw.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("rows "):
            rows = int(line.split()[1])
        elif line.startswith("cols "):
            cols = int(line.split()[1])
        elif line == "matrix":
            in_matrix = True
        elif line.startswith("case "):
            in_matrix = False
            kv = dict(tok.split("=", 1) for tok in line.split()[1:])
            ids = [int(t) for t in kv["ids"].split(",") if t != ""]
            cases.append({"mode": kv["mode"], "ids": ids, "count": int(kv["count"]),
                          "mask": kv["mask"]})
        elif in_matrix:
            matrix.append([float(t) for t in line.split()])
        else:
            raise ValueError(f"{name}: cannot parse {raw!r}")
    m = np.array(matrix, dtype=np.float32)
    assert m.shape == (rows, cols), (name, m.shape, rows, cols)
    for c in cases:
        assert len(c["mask"]) == rows and c["mask"].count("1") == c["count"], (name, c)
    return m, cases


def golden_names():
    return sorted(p.name for p in GOLDEN.glob("hand_*.txt"))


def mask_to_bits(mask_words: np.ndarray, rows: int) -> np.ndarray:
    """uint64 words (row r <-> word r/64, bit r%64) -> bool[rows]; also checks the tail is zero."""
    b = np.unpackbits(np.ascontiguousarray(mask_words).view(np.uint8), bitorder="little")
    assert not b[rows:].any(), "bits >= rows must be zero"
    return b[:rows].astype(bool)


def csr(chromosomes):
    offsets = np.zeros(len(chromosomes) + 1, dtype=np.int32)
    offsets[1:] = np.cumsum([len(c) for c in chromosomes])
    ids = np.array([i for c in chromosomes for i in c], dtype=np.int32)
    return offsets, ids


def brute_force_ok(matrix: np.ndarray, ids, mode_on: bool) -> np.ndarray:
    """Pure-Python loops over rows x pairs (independent of the C oracle and of numpy's >=)."""
    out = np.zeros(matrix.shape[0], dtype=bool)
    for r in range(matrix.shape[0]):
        vals = [float(matrix[r, c]) for c in ids]      # float32 -> double is exact
        ok = True
        for i in range(len(vals) - 1):
            if not (vals[i + 1] >= vals[i]):
                ok = False
        if mode_on:
            for v in vals:
                if math.isnan(v):
                    ok = False
        out[r] = ok
    return out


def numpy_ok(matrix: np.ndarray, ids, mode_on: bool) -> np.ndarray:
    """Library restatement (SURVEY.md 8(c) pin 9): compare >= directly, never diff >= 0."""
    S = matrix[:, np.asarray(ids, dtype=np.int64)]
    ok = (S[:, 1:] >= S[:, :-1]).all(axis=1)
    if mode_on:
        ok &= ~np.isnan(S).any(axis=1)
    return ok


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle
