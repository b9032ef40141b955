"""ebic_read_delimited (comma / tab / semicolon, upper-left corner
optional).  Host-only: runs without a GPU.  The checker is an independent plain-Python restatement
(str.split + numpy float32 parsing); files are written by the test with values whose text round-trips
float32 exactly (repr of the float32), so the comparison is bit-exact."""
from __future__ import annotations

import time

import numpy as np
import pytest

from paper_1807_09932_b200 import binding as B


def write_matrix(path, M, delim, corner, crlf=False, quote_names=False, missing="NA", trailing_newline=True):
    rows, cols = M.shape
    q = '"' if quote_names else ""
    names = [f"{q}s{c}{q}" for c in range(cols)]
    header = ([f"{q}gene{q}"] if corner else []) + names
    eol = "\r\n" if crlf else "\n"
    out = [delim.join(header)]
    for r in range(rows):
        vals = [missing if np.isnan(v) else repr(float(np.float32(v))) if np.isfinite(v) else ("inf" if v > 0 else "-inf")
                for v in M[r]]
        out.append(delim.join([f"{q}g{r}{q}"] + vals))
    text = eol.join(out) + (eol if trailing_newline else "")
    path.write_bytes(text.encode())


def plain_python_reader(path, delim):
    """Independent restatement: split lines and fields, skip names, float32 of every field."""
    lines = [ln.rstrip("\r") for ln in path.read_text().split("\n")]
    lines = [ln for ln in lines if ln.strip()]
    data = []
    for ln in lines[1:]:
        fields = ln.split(delim)[1:]
        row = []
        for f in fields:
            f = f.strip().strip('"')
            row.append(np.float32("nan") if f in ("", "NA", "N/A", "NaN", "nan", "null") else np.float32(f))
        data.append(row)
    return np.array(data, dtype=np.float32)


def sample_matrix(seed, rows, cols):
    rng = np.random.default_rng(seed)
    M = rng.standard_normal((rows, cols)).astype(np.float32)
    M[rng.random(M.shape) < 0.05] = np.float32("nan")
    M[0, 0] = np.float32(1e-41)          # denormal
    M[1 % rows, 0] = np.float32(-0.0)
    M[2 % rows, cols - 1] = np.float32(3.4028235e38)
    M[3 % rows, 1 % cols] = np.float32("inf")
    M[4 % rows, 2 % cols] = np.float32(999.0)
    return M


def same_bits(a, b):
    return a.shape == b.shape and (a.view(np.uint32)[~np.isnan(a)] == b.view(np.uint32)[~np.isnan(b)]).all() \
        and (np.isnan(a) == np.isnan(b)).all()


@pytest.mark.parametrize("delim", [",", "\t", ";"])
@pytest.mark.parametrize("corner", [True, False])
@pytest.mark.parametrize("crlf", [False, True])
def test_reader_matches_plain_python(tmp_path, delim, corner, crlf):
    M = sample_matrix(1, 37, 11)
    p = tmp_path / "m.txt"
    write_matrix(p, M, delim, corner, crlf=crlf, quote_names=crlf, missing="NA" if corner else "")
    for given in (delim, ""):                                   # explicit delimiter and auto-detection
        got = B.ebic_read_delimited(p, given)
        assert got.dtype == np.float32 and got.flags.c_contiguous
        assert same_bits(got, plain_python_reader(p, delim))
        assert same_bits(got, M)                                # and the matrix that was written


def test_reader_edge_shapes(tmp_path):
    p = tmp_path / "m.csv"
    write_matrix(p, sample_matrix(2, 1, 1), ",", True, trailing_newline=False)     # 1 x 1, no final newline
    assert B.ebic_read_delimited(p).shape == (1, 1)
    M = sample_matrix(3, 5, 300)                                                   # wide, like GSE84493's 310 columns
    write_matrix(p, M, ";", False, missing="NaN")
    assert same_bits(B.ebic_read_delimited(p), M)
    p.write_text("a,b\n\nr0,1.5,2\n\n\nr1, 3 ,\"4\"\n")                            # blank lines, blanks, quoted values
    assert (B.ebic_read_delimited(p) == np.array([[1.5, 2], [3, 4]], dtype=np.float32)).all()


@pytest.mark.parametrize("text", [
    "",                                   # empty file
    "g,a,b\n",                            # header only
    "g a b\nr0 1 2\n",                    # no known delimiter
    "g,a,b\nr0,1,2\nr1,1\n",              # ragged line (too few)
    "g,a,b\nr0,1,2\nr1,1,2,3\n",          # ragged line (too many)
    "a\nr0,1,2\n",                        # header and data field counts disagree
    "g,a,b\nr0,1,x\n",                    # not a number
    "g,a,b\nr0,1,2abc\n",                 # trailing junk in a number
])
def test_reader_refuses_malformed_files(tmp_path, text):
    p = tmp_path / "bad.csv"
    p.write_text(text)
    with pytest.raises(B.EbicError) as e:
        B.ebic_read_delimited(p)
    assert e.value.status == B.EBIC_ERR_IO


def test_reader_argument_errors(tmp_path):
    with pytest.raises(B.EbicError) as e:
        B.ebic_read_delimited(tmp_path / "missing.csv")
    assert e.value.status == B.EBIC_ERR_IO
    lib = B.load_library()
    assert lib.ebic_read_delimited(None, b",", None, None, None) == B.EBIC_ERR_ARG
    p = tmp_path / "m.csv"
    p.write_text("g,a\nr,1\n")
    with pytest.raises(B.EbicError) as e:
        B.ebic_read_delimited(p, "|")
    assert e.value.status == B.EBIC_ERR_ARG
    lib.ebic_free_host(None)


def test_reader_throughput(tmp_path, capsys):
    """Measurement: MB/s of text parsed on one host core (reported, not asserted beyond a sanity floor)."""
    M = np.random.default_rng(4).standard_normal((20_000, 64)).astype(np.float32)
    p = tmp_path / "big.tsv"
    write_matrix(p, M, "\t", True)
    size = p.stat().st_size
    t0 = time.perf_counter()
    got = B.ebic_read_delimited(p)
    dt = time.perf_counter() - t0
    assert same_bits(got, M)
    with capsys.disabled():
        print(f"\n[reader] {size / 1e6:.1f} MB, {M.size} values in {dt * 1e3:.0f} ms = {size / dt / 1e6:.0f} MB/s")
    assert size / dt > 5e6
