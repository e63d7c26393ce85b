"""CPU tests (-m "not gpu") of the row-sharded solve's host logic (include/amp_pcg.h "row-sharded solve"; SURVEY.md
section 8(e), 8(f) NEXT-3):

* amp_shard_plan / amp_shard_extract (the product's partition, host code of the C ABI, no CUDA call): contiguous cover,
  slice-aligned boundaries, balance, halo widths = the true column extents, block rows that re-assemble to A;
* a world-size-2 and -3 run over the gloo backend: every rank holds ONE block row from that plan and runs Algorithm 4.1
  with the ORACLE's step functions on its rows; the only cross-rank traffic is the halo of p (sent in the storage
  precision u_z the mat-vec gathers: float16 / float32 / float64 payloads) and three all-reduced scalars per iteration.
  The sharded run must reproduce the one-rank oracle: same iteration count (within 1: the dots are added in another
  order), same switch iterations, the same x to rounding — which pins the partition, the column shift, the halo maps
  and the claim that three 8-byte all-reduces suffice for identical decisions on every rank.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

torch = pytest.importorskip("torch")
sp = pytest.importorskip("scipy.sparse")

from workloads import make_config  # noqa: E402

CASES = [("c2", 12), ("c3", 12), ("c4", 10), ("c1", 24), ("c5", 6000)]


@pytest.fixture(scope="module")
def A():
    from paper_2505_04155_b200 import build as B

    B.build()
    import paper_2505_04155_b200 as A

    return A


@pytest.mark.parametrize("name,size", CASES)
@pytest.mark.parametrize("world", [1, 2, 3, 4])
def test_plan_and_extract(A, name, size, world):
    s = make_config(name, size)
    n = s.n
    plan = A.shard_plan(s.rowptr, s.colidx, world)
    assert len(plan) == world and plan[0].row0 == 0 and plan[-1].row1 == n
    full = sp.csr_matrix((s.vals, s.colidx, s.rowptr), shape=(n, n))
    blocks = []
    for r, sh in enumerate(plan):
        assert sh.row0 < sh.row1 and (r == 0 or sh.row0 == plan[r - 1].row1)
        assert sh.row1 % 32 == 0 or r == world - 1          # whole SELL-32 slices
        assert sh.nnz == s.rowptr[sh.row1] - s.rowptr[sh.row0]
        cols = s.colidx[s.rowptr[sh.row0]:s.rowptr[sh.row1]]
        lo, hi = max(0, sh.row0 - int(cols.min())), max(0, int(cols.max()) - (sh.row1 - 1))
        assert sh.halo_lo == (lo + 7) // 8 * 8 and sh.halo_hi == (hi + 7) // 8 * 8
        assert sh.halo_lo % 8 == 0 and sh.halo_hi % 8 == 0
        if r > 0:
            assert sh.halo_lo <= plan[r - 1].row1 - plan[r - 1].row0
        rp, ci, va = A.shard_extract(s.rowptr, s.colidx, s.vals, sh)
        rows = sh.row1 - sh.row0
        assert rp[0] == 0 and rp[-1] == sh.nnz and len(rp) == rows + 1
        assert ci.min() >= 0 and ci.max() < sh.halo_lo + rows + sh.halo_hi
        # the diagonal of row i sits at column halo_lo + i (what the Jacobi set-up of a block row relies on)
        d = np.array([va[rp[i]:rp[i + 1]][ci[rp[i]:rp[i + 1]] == sh.halo_lo + i].sum() for i in range(0, rows, max(1, rows // 50))])
        assert np.array_equal(d, full.diagonal()[sh.row0:sh.row1:max(1, rows // 50)])
        # shifting the columns back gives exactly the rows of A (same order, same values)
        blocks.append(sp.csr_matrix((va, ci.astype(np.int64) - sh.halo_lo + sh.row0, rp), shape=(rows, n)))
    again = sp.vstack(blocks).tocsr()
    assert (again != full).nnz == 0
    assert np.array_equal(again.indices, full.indices) and np.array_equal(again.data, full.data)
    # balance: no rank has more than its share + one slice of the heaviest rows (+ 25 %)
    cost = [sh.nnz + 4 * (sh.row1 - sh.row0) for sh in plan]
    assert max(cost) <= 1.25 * sum(cost) / world + 32 * (np.diff(s.rowptr).max() + 4)


def test_plan_refuses_a_coupling_that_is_not_banded(A):
    n = 256
    Amat = sp.eye(n, format="lil")
    Amat[0, n - 1] = Amat[n - 1, 0] = 0.5      # periodic coupling: rank 0 needs an entry owned by the last rank
    Amat = Amat.tocsr()
    Amat.sort_indices()
    with pytest.raises(A.AmpPcgError, match="banded"):
        A.shard_plan(Amat.indptr.astype(np.int32), Amat.indices.astype(np.int32), 3)
    assert len(A.shard_plan(Amat.indptr.astype(np.int32), Amat.indices.astype(np.int32), 2)) == 2   # 2 ranks are neighbours
    with pytest.raises(A.AmpPcgError, match="32 rows"):
        A.shard_plan(Amat.indptr.astype(np.int32), Amat.indices.astype(np.int32), 9)


def _full_reach_band(n, seed=5):
    """SPD test matrix whose rows around the rank boundary reach every row of the neighbour rank (a halo as wide as the rank)"""
    rng = np.random.default_rng(seed)
    M = sp.random(n, n, density=0.08, random_state=rng, format="lil")
    for b in range(32, n, 32):   # wherever the planner puts the rank boundary (a multiple of 32):
        M[b - 1, n - 1] = 0.25   # the last row below it reaches the LAST row of the matrix
        M[b, 0] = 0.25           # and the first row above it reaches row 0
    M = (M + M.T).tocsr()
    M = (M + sp.diags(np.asarray(abs(M).sum(axis=1)).ravel() + 1.0)).tocsr()
    M.sort_indices()
    return M


@pytest.mark.parametrize("n", [70, 67, 100])
def test_plan_accepts_a_rounded_halo_inside_the_padded_last_rank(A, n):
    """n not a multiple of 8 with a coupling that reaches the last row: the halo width rounded up to 8 exceeds the last rank's
    row count but not its zero-padded length, which is what the exchange pushes (n = 70: rank 1 has 38 rows, halo 40)"""
    M = _full_reach_band(n)
    rp, ci = M.indptr.astype(np.int32), M.indices.astype(np.int32)
    plan = A.shard_plan(rp, ci, 2)
    assert plan[0].row1 % 32 == 0 and plan[1].row1 == n
    rows0, rows1 = plan[0].row1, n - plan[0].row1
    assert rows1 % 8 != 0
    assert plan[0].halo_hi == (rows1 + 7) // 8 * 8 and plan[0].halo_hi > rows1     # wider than the neighbour's row count
    assert plan[1].halo_lo == rows0 and plan[0].halo_lo == 0 and plan[1].halo_hi == 0
    blocks = []
    for sh in plan:
        r_, c_, v_ = A.shard_extract(rp, ci, M.data, sh)
        assert c_.min() >= 0 and c_.max() < sh.halo_lo + (sh.row1 - sh.row0) + sh.halo_hi
        blocks.append(sp.csr_matrix((v_, c_.astype(np.int64) - sh.halo_lo + sh.row0, r_), shape=(sh.row1 - sh.row0, n)))
    assert (sp.vstack(blocks).tocsr() != M).nnz == 0


# ------------------------------------------------------------------ the sharded loop over gloo, oracle arithmetic ----
def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


_NP_STORE = {0: np.float64, 1: np.float32, 2: np.float16}


def _sharded_oracle_run(rank, world, port, name, size, pol_kw, out_dir):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import oracle as O
    import paper_2505_04155_b200 as A

    torch.set_num_threads(1)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s = make_config(name, size)
    plan = A.shard_plan(s.rowptr, s.colidx, world)
    sh = plan[rank]
    rp, ci, va = A.shard_extract(s.rowptr, s.colidx, s.vals, sh)
    n, hlo, hhi = sh.row1 - sh.row0, sh.halo_lo, sh.halo_hi
    send_lo = plan[rank - 1].halo_hi if rank > 0 else 0           # what my neighbours need from me
    send_hi = plan[rank + 1].halo_lo if rank + 1 < world else 0
    b = s.b[sh.row0:sh.row1].copy()
    pol = O.make_policy(**pol_kw)
    tol, maxit = s.tol, s.maxit
    diag = np.array([va[rp[i]:rp[i + 1]][ci[rp[i]:rp[i + 1]] == hlo + i].sum() for i in range(n)])
    dinv = 1.0 / diag
    dinv32 = dinv.astype(np.float32).astype(np.float64)
    va32 = va  # O.spmv_fp32 rounds the values itself

    def allsum(v):
        t = torch.tensor([v], dtype=torch.float64)
        parts = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(parts, t)            # every rank adds ALL partial sums in rank order: identical scalars everywhere
        tot = 0.0
        for p_ in parts:
            tot += float(p_[0])
        return tot

    sent_bytes = []

    def exchange(p_loc, prec):
        """halo of p in the storage precision the mat-vec gathers; returns the extended vector [halo_lo | owned | halo_hi]"""
        dt = _NP_STORE[prec]
        ext = np.zeros(hlo + n + hhi, dtype=np.float64)
        ext[hlo:hlo + n] = p_loc
        reqs, bufs = [], {}
        if rank > 0:
            if send_lo:
                t = torch.from_numpy(p_loc[:send_lo].astype(dt)); sent_bytes.append(t.numel() * t.element_size())
                assert np.array_equal(t.numpy().astype(np.float64), p_loc[:send_lo])      # stored values travel exactly
                reqs.append(dist.isend(t, rank - 1))
            if hlo:
                bufs["lo"] = torch.empty(hlo, dtype=torch.from_numpy(np.zeros(1, dtype=dt)).dtype)
                reqs.append(dist.irecv(bufs["lo"], rank - 1))
        if rank + 1 < world:
            if send_hi:
                t = torch.from_numpy(p_loc[n - send_hi:].astype(dt)); sent_bytes.append(t.numel() * t.element_size())
                reqs.append(dist.isend(t, rank + 1))
            if hhi:
                bufs["hi"] = torch.empty(hhi, dtype=torch.from_numpy(np.zeros(1, dtype=dt)).dtype)
                reqs.append(dist.irecv(bufs["hi"], rank + 1))
        for q_ in reqs:
            q_.wait()
        if "lo" in bufs:
            ext[:hlo] = bufs["lo"].numpy().astype(np.float64)
        if "hi" in bufs:
            ext[hlo + n:] = bufs["hi"].numpy().astype(np.float64)
        return ext

    # Algorithm 4.1 on this rank's rows, step by step as oracle/amp_pcg_oracle.cpp does it (x0 = 0: r0 = b)
    x = np.zeros(n); r = b.copy(); p = np.zeros(n)
    nb = np.sqrt(allsum(O.dot(b, b)))
    delta = np.sqrt(allsum(O.dot(r, r)))
    hist = np.zeros(maxit + 2); hist[0] = delta
    ur, uz = O.FP64, (pol.u0 if pol.amp else O.FP64)
    it_ur32 = it_uz32 = it_uz16 = -1
    rho_prev, status, k = 0.0, 1, 0
    halo_precs = []
    for k in range(maxit):
        if pol.amp:
            if ur == O.FP64 and O.eta(pol, hist, k) <= pol.eta_safety * tol * nb:
                ur, it_ur32 = O.FP32, k
                r = O.round_fp32(r)
            want = O.select_uz(pol, delta / nb)
            if want > uz:
                uz = want
                if uz >= O.FP32 and it_uz32 < 0: it_uz32 = k
                if uz == O.FP16 and it_uz16 < 0: it_uz16 = k
                p = O.round_fp16(p) if uz == O.FP16 else O.round_fp32(p)
        omega = 1.0 / delta if pol.amp else 1.0
        z, _ = O.step_z(r, omega, dinv if uz == O.FP64 else dinv32, ur, uz)
        rho = allsum(O.dot(r, z))
        beta = rho / rho_prev if k > 0 else 0.0
        p, _ = O.step_p(beta, p, z, uz)
        gather_prec = O.FP32 if (uz == O.FP64 and ur == O.FP32) else uz     # RN32(p) while u_z = FP64 and u_r = FP32
        halo_precs.append(gather_prec)
        pg = O.round_fp32(p) if gather_prec != uz else p
        ext = exchange(pg, gather_prec)
        q = O.spmv_fp64(rp, ci, va, ext) if ur == O.FP64 else O.spmv_fp32(rp, ci, va32, ext)
        gamma = allsum(O.dot(q, p))
        if not (gamma > 0.0 and rho > 0.0):
            status = -2
            break
        alpha = rho / gamma
        x, r = O.step_xr(alpha, p, q, x, r, ur)
        delta = np.sqrt(allsum(O.dot(r, r)))
        hist[k + 1] = delta
        rho_prev = rho
        if delta <= pol.stop_safety * tol * nb:
            status, k = 0, k + 1
            break
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), x=x, iters=k, status=status, sw=np.array([it_ur32, it_uz32, it_uz16]),
             row0=sh.row0, row1=sh.row1, halo_precs=np.array(halo_precs), sent=np.array(sent_bytes), hist=hist[:k + 1],
             counts=np.array([send_lo, send_hi]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("name,size,world,pol_kw", [
    ("c2", 12, 2, dict(amp=1, u0=0, eta_rule=0)),
    ("c3", 12, 2, dict(amp=1, u0=0, eta_rule=0)),
    ("c3", 12, 3, dict(amp=1, u0=2, eta_rule=1)),
    ("c5", 6000, 2, dict(amp=1, u0=0, eta_rule=0)),
    ("c2", 12, 2, dict(amp=0)),
])
def test_sharded_run_over_gloo_reproduces_the_one_rank_oracle(A, tmp_path, name, size, world, pol_kw):
    import torch.multiprocessing as mp

    import oracle as O

    s = make_config(name, size)
    ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(**pol_kw))
    mp.spawn(_sharded_oracle_run, args=(world, _free_port(), name, size, pol_kw, str(tmp_path)), nprocs=world, join=True)
    outs = [np.load(tmp_path / f"r{r}.npz") for r in range(world)]
    x = np.concatenate([o["x"] for o in outs])
    for o in outs:  # every rank took the same decisions
        assert int(o["status"]) == ref.status == 0
        assert int(o["iters"]) == int(outs[0]["iters"]) and np.array_equal(o["sw"], outs[0]["sw"])
        assert np.array_equal(o["hist"], outs[0]["hist"])           # bit-identical scalars on all ranks
    assert abs(int(outs[0]["iters"]) - ref.iters) <= 1
    assert np.array_equal(outs[0]["sw"], [ref.it_ur32, ref.it_uz32, ref.it_uz16])
    assert np.allclose(outs[0]["hist"][:20], ref.hist[:20], rtol=1e-9)
    assert np.linalg.norm(x - ref.x) <= 1e-6 * np.linalg.norm(ref.x)
    A_ = sp.csr_matrix((s.vals, s.colidx, s.rowptr), shape=(s.n, s.n))
    assert np.linalg.norm(s.b - A_ @ x) <= 2 * s.tol * np.linalg.norm(s.b)
    # the halo shrinks with the precision: bytes per exchange = entries x (8, 4, 2)
    o = outs[0]
    per = int(o["counts"].sum())
    if per and pol_kw.get("amp"):
        sizes = {0: 8, 1: 4, 2: 2}
        expect = sum(sizes[int(pc)] for pc in o["halo_precs"]) * per
        assert int(o["sent"].sum()) == expect
        if pol_kw.get("u0") == 2:
            assert set(o["halo_precs"].tolist()) == {2}            # AMP-PCG(FP16): FP16 halos throughout
        else:
            assert o["halo_precs"][-1] == 2 and o["halo_precs"][0] == 0


@pytest.mark.parametrize("name", ["c2", "c5"])
def test_plan_at_full_size_for_eight_ranks(A, name):
    """the partition bench.py --shard would use on the real configs: 8 ranks, halo = one grid plane (c2) / the 50 000-row
    band (c5), balanced to a few per cent"""
    s = make_config(name)
    plan = A.shard_plan(s.rowptr, s.colidx, 8)
    rows = [sh.row1 - sh.row0 for sh in plan]
    cost = [sh.nnz + 4 * r for sh, r in zip(plan, rows)]
    assert max(cost) <= 1.03 * sum(cost) / 8
    halo = max(max(sh.halo_lo, sh.halo_hi) for sh in plan)
    if name == "c2":
        assert halo == 128 * 128 and all(sh.halo_lo in (0, halo) and sh.halo_hi in (0, halo) for sh in plan)
    else:
        assert 49000 <= halo <= 50008 and halo < min(rows)
    # bytes per iteration that cross ranks, FP16 phase: 2 B per halo entry (the 4x shrink against FP64 is AMP's)
    assert sum(sh.halo_lo + sh.halo_hi for sh in plan) * 2 <= (2 * 7 * halo) * 2
