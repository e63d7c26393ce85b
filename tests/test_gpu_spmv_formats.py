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

amp_create_opts_t.index_format (AMP_INDEX_NO_ALIGN / AMP_INDEX_FORCE32) forces the more general formats on
the same matrix, so every kernel path sees every matrix class.
"""
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


def _check_bitwise(rowptr, colidx, vals, n, expect_bytes_per_entry=None, **opts):
    rng = np.random.default_rng(3)
    p = rng.standard_normal(n)
    npad = (n + 7) // 8 * 8
    p16 = np.zeros(npad, dtype=np.float16)
    p16[:n] = p.astype(np.float16)
    dev = [torch.from_numpy(a).cuda() for a in (rowptr, colidx, vals)]
    with A.AmpPcg(*dev, A.PRECOND_NONE, **opts) as h:
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


@pytest.mark.parametrize("name,size", [("c1", 37), ("c2", 19), ("c3", 21), ("c4", 17)])
@pytest.mark.parametrize("fmt", [A.INDEX_AUTO, A.INDEX_NO_ALIGN, A.INDEX_FORCE32])
@pytest.mark.parametrize("kernel", [A.SPMV_DIRECT, A.SPMV_PIPELINED])
def test_stencils_in_every_format(name, size, fmt, kernel):
    s = make_config(name, size)
    if kernel == A.SPMV_PIPELINED and fmt != A.INDEX_AUTO:
        # the bulk-copy pipelined kernel exists for diagonal-aligned slices only: asking for it on another format is an error
        with pytest.raises(A.AmpPcgError):
            A.AmpPcg(*[torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals)], A.PRECOND_NONE, index_format=fmt,
                     spmv_kernel=kernel)
        return
    if kernel == A.SPMV_PIPELINED:
        # every slice must be diagonal-aligned: take grid edges that are multiples of the slice height
        s = make_config(name, {"c1": 96, "c2": 32, "c3": 32, "c4": 32}[name])
    # FP32 phase: 4 B value + index bytes per stored entry (padding included, so a little above the nominal)
    expect = {A.INDEX_AUTO: (4.0, 4.9), A.INDEX_NO_ALIGN: (6.0, 7.2), A.INDEX_FORCE32: (8.0, 9.3)}[fmt]
    _check_bitwise(s.rowptr, s.colidx, s.vals, s.n, expect, index_format=fmt, spmv_kernel=kernel)


def test_banded_scattered_uses_16_bit_offsets():
    n = 20011
    rowptr, colidx, vals = _banded_scattered(n, 3000, 9, 11)
    per_entry = _check_bitwise(rowptr, colidx, vals, n)
    assert per_entry < 7.5  # 4 B value + 2 B offset + bases + padding: well below the 8+ B of 32-bit indices
    assert _check_bitwise(rowptr, colidx, vals, n, index_format=A.INDEX_FORCE32) >= 8.0


def test_wide_pattern_falls_back_to_32_bit_indices():
    n = 150001  # offsets up to +-70000 from the diagonal: do not fit 16 bits
    rowptr, colidx, vals = _banded_scattered(n, 70000, 11, 12)
    assert _check_bitwise(rowptr, colidx, vals, n) >= 8.0


def test_varying_row_lengths_are_sorted_into_slices():
    n = 9973
    rowptr, colidx, vals = _varying_lengths(n, 13)
    per_entry = _check_bitwise(rowptr, colidx, vals, n)
    # unsorted, a slice is as wide as its longest row (about 2x the mean here); sorted, padding is a few percent
    assert per_entry < 9.5


def test_c5_like_random_spd():
    s = make_config("c5", 30000)
    _check_bitwise(s.rowptr, s.colidx, s.vals, s.n)


def test_long_rows_next_to_aligned_slices():
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


def test_long_rows_at_high_indices_of_a_large_irregular_matrix():
    # Rows longer than the slice cap keep a zero-length slot in their slice; the block that sums them from the CSR
    # arrays must be the ONLY writer of their q.  With n >= 2 M and an irregular pattern the grid has several waves, so
    # a slice-owning block can run long after the long-row block: any store from the slice loop would overwrite q with 0.
    import scipy.sparse as sp

    n = 2_100_003
    rng = np.random.default_rng(77)
    lens = rng.integers(0, 10, n)
    rows = np.repeat(np.arange(n), lens)
    cols = rng.integers(0, n, rows.size)
    longs = np.array([n - 1, n - 1000, n - 31, n // 2 + 7, 3])
    lr = np.repeat(longs, 5000)
    lc = rng.integers(0, n, lr.size)
    R = sp.coo_matrix((rng.standard_normal(rows.size + lr.size), (np.concatenate([rows, lr]), np.concatenate([cols, lc]))),
                      shape=(n, n)).tocsr()
    S = (R + R.T).tocsr()
    dg = np.asarray(abs(S).sum(axis=1)).ravel() + 1.0
    Aspd = (S + sp.diags(dg)).tocsr()
    Aspd.sum_duplicates(); Aspd.sort_indices()
    rowptr, colidx, vals = Aspd.indptr.astype(np.int32), Aspd.indices.astype(np.int32), Aspd.data.astype(np.float64)
    rl = np.diff(rowptr)
    assert (rl[longs] > 4000).all()
    p = rng.standard_normal(n)
    b = rng.standard_normal(n)
    dev = [torch.from_numpy(a).cuda() for a in (rowptr, colidx, vals)]
    absAp = abs(Aspd) @ np.abs(p)
    short = np.ones(n, dtype=bool)
    short[rl > max(256, 8 * int(np.ceil(len(colidx) / n)))] = False
    assert (~short).sum() >= len(longs)
    ref64 = O.spmv_fp64(rowptr, colidx, vals, p)
    p16 = np.zeros((n + 7) // 8 * 8, dtype=np.float16); p16[:n] = p.astype(np.float16)
    ref32 = O.spmv_fp32(rowptr, colidx, vals, p16[:n].astype(np.float64))
    with A.AmpPcg(*dev, A.PRECOND_JACOBI) as h:
        for _ in range(3):  # the race was timing dependent
            q = h.spmv(torch.from_numpy(p).cuda(), A.FP64).cpu().numpy()
            assert np.array_equal(q[short], ref64[short])
            assert np.all(np.abs(q - ref64) <= 6000 * 2.0 ** -53 * absAp + 1e-300)
            assert np.all(q[longs] != 0.0)
            q32 = h.spmv(torch.from_numpy(p16).cuda(), A.FP32).cpu().numpy().astype(np.float64)
            assert np.array_equal(q32[short], ref32[short])
            assert np.all(np.abs(q32 - ref32) <= 2 * 6000 * 2.0 ** -24 * (abs(Aspd) @ np.abs(p16[:n].astype(np.float64))) + 1e-30)
        # the in-loop kernel, in all three loop drivers: the first iterations track the oracle's
        for spec in (dict(amp=0), dict(amp=1, u0=2, eta_rule=1, eps32=1e-30)):
            ref = O.amp_pcg(rowptr, colidx, vals, b, 1e-30, 8, O.make_policy(**spec))
            for loop in (A.LOOP_STREAM, A.LOOP_GRAPH, A.LOOP_PERSISTENT):
                x = torch.zeros(n, dtype=torch.float64, device="cuda")
                st = h.solve(torch.from_numpy(b).cuda(), x, 1e-30, 8, A.Policy.default(x0_zero=1, loop_mode=loop, **spec))
                assert st.iters == 8
                assert np.allclose(h.residual_history(), ref.hist, rtol=1e-6), (spec, loop)


def test_format_info_reports_what_create_built():
    """amp_pcg_format_info: structured-grid matrices are diagonal-aligned throughout; narrow stencils (c1-c3) mark nearly
    all slices as the uniform stencil (columns = row + a constant; boundary slices of the grid lack diagonals and keep the
    general aligned path); c4 runs the pipelined mat-vec; c5 has sorted rows and 16-bit offsets."""
    def info(name, size, **opts):
        s = make_config(name, size)
        with A.AmpPcg(*[torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals)], **opts) as h:
            return s, h.format_info()

    for name, size, w, maxoff in (("c1", 64, 5, 64), ("c2", 64, 7, 64 * 64), ("c3", 64, 7, 64 * 64)):
        s, fi = info(name, size)
        assert fi.slices == (s.n + 31) // 32 and fi.aligned_slices == fi.slices and fi.index_bits == 0, fi.asdict()
        assert fi.uniform_width == w and fi.uniform_slices >= 0.9 * fi.slices, fi.asdict()
        assert fi.guard >= maxoff and fi.long_rows == 0 and fi.rows_sorted == 0, fi.asdict()
        assert fi.stored_entries >= s.nnz
        _, fi2 = info(name, size, index_format=A.INDEX_NO_ALIGN)
        assert fi2.aligned_slices == 0 and fi2.uniform_slices == 0 and fi2.index_bits == 16
    s, fi = info("c4", 32)
    assert fi.aligned_slices == fi.slices and fi.spmv_pipelined == 1 and fi.uniform_slices == 0   # 27 entries per row: not narrow
    s, fi = info("c5", 30000)
    assert fi.aligned_slices == 0 and fi.rows_sorted == 1 and fi.index_bits == 16
    s, fi = info("c2", 24, vec_kernel=A.VEC_STAGED)
    assert fi.vec_staged == 3
