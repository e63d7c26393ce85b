"""-m gpu: every storage mode of the SELL-32 repack (csrc/spmv.cuh) against the oracle's CSR mat-vec.

The library keeps the entries of a row in CSR order and accumulates ONE fma chain per row in the
working precision, which is exactly what the oracle's spmv_fp64 / spmv_fp32 do, so
for rows that live in the slices the results must be BIT-IDENTICAL in both precisions, whatever index
format create() picked:

* diagonal-aligned slices (implicit columns)           — stencil matrices,
* 16-bit column offsets from a per-(slice, entry) base — banded matrices with scattered columns,
* 32-bit column indices                                — wide / random patterns,
* row order sorted by length inside windows            — strongly varying row lengths,
* rows longer than the slice cap (summed from the CSR arrays by a whole block: tolerance, not bits).

The environment variables AMP_SPMV_NO_ALIGN / AMP_SPMV_IDX32 (tuning aids read by amp_pcg_create)
force the more general formats on the same matrix, so every kernel path sees every matrix class.
"""
import os

import numpy as np
import pytest

import oracle as O
from workloads import make_config

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")


def _csr_from_rows(rows, n, rng, diag=True):
    cols, lens = [], []
    for i, r in enumerate(rows):
        r = np.unique(np.concatenate([r, [i]]) if diag else r)  # sorted, no duplicates
        cols.append(r)
        lens.append(len(r))
    rowptr = np.zeros(n + 1, dtype=np.int32)
    rowptr[1:] = np.cumsum(lens)
    colidx = np.concatenate(cols).astype(np.int32)
    vals = rng.standard_normal(len(colidx))
    return rowptr, colidx, vals


def _banded_scattered(n, band, per_row, seed):
    """random columns within +-band of the diagonal: not diagonal-aligned, offsets fit 16 bits if band < 32768"""
    rng = np.random.default_rng(seed)
    rows = [np.clip(i + rng.integers(-band, band + 1, per_row), 0, n - 1) for i in range(n)]
    return _csr_from_rows(rows, n, rng)


def _varying_lengths(n, seed):
    rng = np.random.default_rng(seed)
    rows = [rng.integers(0, n, int(rng.integers(0, 40))) for _ in range(n)]
    return _csr_from_rows(rows, n, rng, diag=False)


def _check_bitwise(rowptr, colidx, vals, n, expect_bytes_per_entry=None):
    rng = np.random.default_rng(3)
    p = rng.standard_normal(n)
    npad = (n + 7) // 8 * 8
    p16 = np.zeros(npad, dtype=np.float16)
    p16[:n] = p.astype(np.float16)
    dev = [torch.from_numpy(a).cuda() for a in (rowptr, colidx, vals)]
    with A.AmpPcg(*dev, A.PRECOND_NONE) as h:
        q = h.spmv(torch.from_numpy(p).cuda(), A.FP64).cpu().numpy()
        ref = O.spmv_fp64(rowptr, colidx, vals, p)
        assert np.array_equal(q, ref), float(np.max(np.abs(q - ref)))
        q32 = h.spmv(torch.from_numpy(p16).cuda(), A.FP32).cpu().numpy()
        ref32 = O.spmv_fp32(rowptr, colidx, vals, p16[:n].astype(np.float64)).astype(np.float32)
        assert np.array_equal(q32, ref32), float(np.max(np.abs(q32.astype(np.float64) - ref32)))
        bytes32 = h.spmv_bytes(A.FP32, A.FP16)
    nnz = len(colidx)
    per_entry = (bytes32 - n * 6.0) / max(nnz, 1)
    if expect_bytes_per_entry is not None:
        lo, hi = expect_bytes_per_entry
        assert lo <= per_entry <= hi, per_entry
    return per_entry


@pytest.fixture
def clean_env():
    saved = {k: os.environ.pop(k, None) for k in ("AMP_SPMV_NO_ALIGN", "AMP_SPMV_IDX32")}
    yield
    for k, v in saved.items():
        os.environ.pop(k, None)
        if v is not None:
            os.environ[k] = v


@pytest.mark.parametrize("name,size", [("c1", 37), ("c2", 19), ("c3", 21), ("c4", 17)])
@pytest.mark.parametrize("force", ["", "AMP_SPMV_NO_ALIGN", "AMP_SPMV_NO_ALIGN+AMP_SPMV_IDX32"])
def test_stencils_in_every_format(clean_env, name, size, force):
    s = make_config(name, size)
    for k in filter(None, force.split("+")):
        os.environ[k] = "1"
    # FP32 phase: 4 B value + index bytes per stored entry (padding included, so a little above the nominal)
    expect = {"": (4.0, 4.9), "AMP_SPMV_NO_ALIGN": (6.0, 7.2), "AMP_SPMV_NO_ALIGN+AMP_SPMV_IDX32": (8.0, 9.3)}[force]
    _check_bitwise(s.rowptr, s.colidx, s.vals, s.n, expect)


def test_banded_scattered_uses_16_bit_offsets(clean_env):
    n = 20011
    rowptr, colidx, vals = _banded_scattered(n, 3000, 9, 11)
    per_entry = _check_bitwise(rowptr, colidx, vals, n)
    assert per_entry < 7.5  # 4 B value + 2 B offset + bases + padding: well below the 8+ B of 32-bit indices
    os.environ["AMP_SPMV_IDX32"] = "1"
    assert _check_bitwise(rowptr, colidx, vals, n) >= 8.0


def test_wide_pattern_falls_back_to_32_bit_indices(clean_env):
    n = 150001  # offsets up to +-70000 from the diagonal: do not fit 16 bits
    rowptr, colidx, vals = _banded_scattered(n, 70000, 11, 12)
    assert _check_bitwise(rowptr, colidx, vals, n) >= 8.0


def test_varying_row_lengths_are_sorted_into_slices(clean_env):
    n = 9973
    rowptr, colidx, vals = _varying_lengths(n, 13)
    per_entry = _check_bitwise(rowptr, colidx, vals, n)
    # unsorted, a slice is as wide as its longest row (about 2x the mean here); sorted, padding is a few percent
    assert per_entry < 9.5


def test_c5_like_random_spd(clean_env):
    s = make_config("c5", 30000)
    _check_bitwise(s.rowptr, s.colidx, s.vals, s.n)


def test_long_rows_next_to_aligned_slices(clean_env):
    # 2-D stencil plus two dense rows (longer than the slice cap): they are summed from the CSR arrays
    s = make_config("c1", 40)
    n = s.n
    rows = [s.colidx[s.rowptr[i]:s.rowptr[i + 1]].astype(np.int64) for i in range(n)]
    rows[5] = np.arange(n)
    rows[n - 7] = np.arange(0, n, 2)
    rng = np.random.default_rng(5)
    rowptr, colidx, vals = _csr_from_rows(rows, n, rng)
    p = rng.standard_normal(n)
    dev = [torch.from_numpy(a).cuda() for a in (rowptr, colidx, vals)]
    with A.AmpPcg(*dev, A.PRECOND_NONE) as h:
        q = h.spmv(torch.from_numpy(p).cuda(), A.FP64).cpu().numpy()
    ref = O.spmv_fp64(rowptr, colidx, vals, p)
    short = np.ones(n, dtype=bool)
    short[[5, n - 7]] = False
    assert np.array_equal(q[short], ref[short])
    import scipy.sparse as sp
    absAp = sp.csr_matrix((np.abs(vals), colidx, rowptr), shape=(n, n)) @ np.abs(p)
    assert np.all(np.abs(q - ref) <= n * 2.0 ** -53 * absAp)
