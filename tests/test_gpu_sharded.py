"""-m gpu: the row-sharded solve (include/amp_pcg.h "row-sharded solve") on ONE GPU.

All ranks of a group are driven by this process on one device and one stream (amp_pcg_shard_attach_local): the kernels
are the ones a multi-GPU run launches — peer stores of the halo of p into the neighbour's band, flags, mailbox posts,
k_epi — only the concurrency is missing (a kernel that waits for a peer finds that the peer has already run), which
is the emulation the profiling recipe prescribes for fewer GPUs than ranks.

* amp_spmv_sharded: q is BIT-IDENTICAL to the unsharded mat-vec (same fma chain per row), every precision pairing;
* amp_pcg_solve_sharded against the oracle and against the unsharded solve of this library: iteration count within 1
  (the inner products are added per rank, then in rank order), switch iterations within 1, true residual <= 2 tol
  (<= tol strict), x to 1e-6; identical results on every rank by construction (the call fails if ranks disagree).
"""
import numpy as np
import pytest

from workloads import make_config
from gpu_util import POLICY_SPECS, cuda_policy, iters_close, oracle_policy, switch_close, to_device

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")
O = pytest.importorskip("oracle")


def make_group(s, world, **opts):
    plan = A.shard_plan(s.rowptr, s.colidx, world)
    handles, parts = [], []
    for sh in plan:
        rp, ci, va = A.shard_extract(s.rowptr, s.colidx, s.vals, sh)
        t = [torch.from_numpy(a).cuda() for a in (rp, ci, va)]
        handles.append(A.AmpPcg(*t, A.PRECOND_JACOBI, halo_lo=sh.halo_lo, halo_hi=sh.halo_hi, **opts))
        parts.append((int(sh.row0), int(sh.row1)))
    return A.ShardGroup.attach_local(handles), parts


def split(v, parts):
    return [v[a:b].contiguous() for a, b in parts]


@pytest.mark.parametrize("name,size", [("c2", 20), ("c3", 18), ("c4", 24), ("c5", 40000), ("c1", 40)])
@pytest.mark.parametrize("world", [1, 2, 3, 4])
def test_sharded_spmv_is_bit_identical(name, size, world):
    s = make_config(name, size)
    rp, ci, va, _ = to_device(s)
    rng = np.random.default_rng(11)
    p64 = torch.from_numpy(rng.uniform(-1, 1, s.n)).cuda()
    g, parts = make_group(s, world)
    try:
        with A.AmpPcg(rp, ci, va) as whole:
            for vec_dt in (torch.float64, torch.float32, torch.float16):
                p = p64.to(vec_dt)
                for mat in (A.FP64, A.FP32):
                    if vec_dt == torch.float16:
                        npad = (s.n + 7) // 8 * 8
                        pw = torch.zeros(npad, dtype=vec_dt, device="cuda"); pw[:s.n] = p
                    else:
                        pw = p
                    q_ref = whole.spmv(pw, mat)
                    q = torch.cat(g.spmv(split(p, parts), mat))
                    assert torch.equal(q, q_ref), (vec_dt, mat)
            qo = O.spmv_fp64(s.rowptr, s.colidx, s.vals, p64.cpu().numpy())
            assert np.array_equal(torch.cat(g.spmv(split(p64, parts), A.FP64)).cpu().numpy(), qo)
    finally:
        g.close()


SOLVE_POLICIES = ["pcg_fp64", "amp_fp64_delay", "amp_fp16_linear", "amp_fp64_delay_strict", "amp_fp64_delay_lagged", "amp_fp64_delay_rms"]


@pytest.mark.parametrize("name,size", [("c2", 20), ("c3", 18), ("c4", 24), ("c5", 40000)])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_sharded_solve_matches_oracle_and_unsharded(name, size, world):
    s = make_config(name, size)
    rp, ci, va, b = to_device(s)
    g, parts = make_group(s, world)
    crow = rp.to(torch.int64)
    At = torch.sparse_csr_tensor(crow, ci.to(torch.int64), va, size=(s.n, s.n))
    bn = float(torch.linalg.norm(b))
    try:
        with A.AmpPcg(rp, ci, va) as whole:
            for pname in SOLVE_POLICIES:
                spec = POLICY_SPECS[pname]
                ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec))
                x1 = torch.zeros(s.n, dtype=torch.float64, device="cuda")
                st1 = whole.solve(b, x1, s.tol, s.maxit, cuda_policy(spec, x0_zero=1))
                modes = [A.LOOP_AUTO] + ([A.LOOP_STREAM] if world == 1 else [])   # world 1: graph (AUTO) and stream
                for lm in modes:
                    xs = [torch.zeros(bb - aa, dtype=torch.float64, device="cuda") for aa, bb in parts]
                    sts = g.solve(split(b, parts), xs, s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=lm))
                    x = torch.cat(xs)
                    st = sts[0]
                    assert all((t.status, t.iters, t.it_ur32, t.it_uz32, t.it_uz16) ==
                               (st.status, st.iters, st.it_ur32, st.it_uz32, st.it_uz16) for t in sts)
                    assert st.status == ref.status == 0, (pname, st.status)
                    assert st.loop_mode == (A.LOOP_GRAPH if (world == 1 and lm == A.LOOP_AUTO) else A.LOOP_STREAM)
                    assert abs(st.iters - st1.iters) <= 1 and iters_close(st.iters, ref.iters), (pname, st.iters, st1.iters, ref.iters)
                    for key in ("it_ur32", "it_uz32", "it_uz16"):
                        assert switch_close(getattr(st, key), getattr(ref, key), 1), (pname, key, getattr(st, key), getattr(ref, key))
                    true = float(torch.linalg.norm(b - At @ x)) / bn
                    assert st.relres_true == pytest.approx(true, rel=1e-5)
                    assert true <= (1.0 if spec.get("eta_safety", 1.0) < 1.0 else 2.0) * s.tol, (pname, true)
                    assert float(torch.linalg.norm(x - x1)) <= 1e-6 * float(torch.linalg.norm(x1))
    finally:
        g.close()


def test_sharded_solve_with_staged_vector_kernels():
    """the bulk-copy staged z / x-r kernels post their partial sums to the mailboxes like the direct ones"""
    s = make_config("c3", 18)
    rp, ci, va, b = to_device(s)
    g, parts = make_group(s, 3, vec_kernel=A.VEC_STAGED)
    try:
        assert all(h.format_info().vec_staged == 3 for h in g.handles)
        for pname in ("amp_fp64_delay", "amp_fp64_delay_lagged", "pcg_fp64"):
            spec = POLICY_SPECS[pname]
            ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec))
            xs = [torch.zeros(bb - aa, dtype=torch.float64, device="cuda") for aa, bb in parts]
            st = g.solve(split(b, parts), xs, s.tol, s.maxit, cuda_policy(spec, x0_zero=1))[0]
            assert st.status == 0 and iters_close(st.iters, ref.iters) and st.relres_true <= 2 * s.tol
            for key in ("it_ur32", "it_uz32", "it_uz16"):
                assert switch_close(getattr(st, key), getattr(ref, key), 1)
    finally:
        g.close()


def test_sharded_edge_cases():
    s = make_config("c3", 16)
    rp, ci, va, b = to_device(s)
    g, parts = make_group(s, 3)
    try:
        spec = POLICY_SPECS["amp_fp64_delay"]
        # x0 != 0: r0 = b - A x0 needs the halo of x0
        rng = np.random.default_rng(5)
        x0 = torch.from_numpy(rng.uniform(-1, 1, s.n)).cuda()
        ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec), x0=x0.cpu().numpy())
        xs = [t.clone() for t in split(x0, parts)]
        sts = g.solve(split(b, parts), xs, s.tol, s.maxit, cuda_policy(spec))
        assert sts[0].status == 0 and abs(sts[0].iters - ref.iters) <= 1
        assert sts[0].relres_true <= 2 * s.tol
        hist = g.handles[0].residual_history()
        assert hist[0] == pytest.approx(ref.hist[0], rel=1e-13)
        # b = 0: x = 0, 0 iterations
        xs = [t.clone() for t in split(x0, parts)]
        zb = [torch.zeros_like(t) for t in split(b, parts)]
        sts = g.solve(zb, xs, s.tol, s.maxit, cuda_policy(spec))
        assert sts[0].status == 0 and sts[0].iters == 0 and all(float(t.abs().max()) == 0.0 for t in xs)
        # maxit
        xs = [torch.zeros_like(t) for t in split(b, parts)]
        sts = g.solve(split(b, parts), xs, s.tol, 7, cuda_policy(spec, x0_zero=1))
        assert sts[0].status == 1 and sts[0].iters == 7
        # a block row is not a system of its own
        with pytest.raises(A.AmpPcgError, match="sharded"):
            g.handles[1].solve(split(b, parts)[1], xs[1], s.tol, 5)
        with pytest.raises(A.AmpPcgError, match="sharded"):
            g.handles[1].spmv(xs[1])
        with pytest.raises(A.AmpPcgError):   # persistent loop is not available
            g.solve(split(b, parts), xs, s.tol, 5, cuda_policy(spec, loop_mode=A.LOOP_PERSISTENT))
    finally:
        g.close()


def test_attach_refuses_inconsistent_halos():
    s = make_config("c2", 16)
    plan = A.shard_plan(s.rowptr, s.colidx, 2)
    hs = []
    for i, sh in enumerate(plan):
        rp, ci, va = A.shard_extract(s.rowptr, s.colidx, s.vals, sh)
        t = [torch.from_numpy(a).cuda() for a in (rp, ci, va)]
        hs.append(A.AmpPcg(*t, A.PRECOND_JACOBI, halo_lo=sh.halo_lo, halo_hi=sh.halo_hi))
    with pytest.raises(A.AmpPcgError):
        A.ShardGroup.attach_local(hs[::-1])     # rank order reversed: rank 0 would have a lower halo
    g = A.ShardGroup.attach_local(hs)
    g.close()


def test_export_blob_describes_the_rank():
    s = make_config("c2", 16)
    g, parts = make_group(s, 2)
    try:
        e = A.ShardExport.from_buffer_copy(A.ShardGroup.export(g.handles[1]))
        assert e.n == parts[1][1] - parts[1][0] and e.halo_lo == 256 and e.halo_hi == 0   # one 16 x 16 plane
        assert e.guard >= e.halo_lo and e.off[1] == 8 * e.guard and e.off[3] == 2 * e.guard
        assert any(bytes(e.mem[0])) and any(bytes(e.mem[3]))
    finally:
        g.close()


def test_attach_through_export_blobs_single_rank():
    """amp_pcg_shard_export / amp_pcg_shard_attach with a group of one (no peer to open): the one-process-per-GPU wiring,
    whose reducing kernels collect and step inline and whose loop is the WHILE-node graph"""
    s = make_config("c3", 18)
    rp, ci, va, b = to_device(s)
    spec = POLICY_SPECS["amp_fp64_delay"]
    ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec))
    h = A.AmpPcg(rp, ci, va)
    g = A.ShardGroup.attach_ipc(h, 0, [A.ShardGroup.export(h)])
    try:
        for lm in (A.LOOP_AUTO, A.LOOP_STREAM):
            x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
            st = g.solve([b], [x], s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=lm))[0]
            assert st.status == 0 and st.loop_mode == (A.LOOP_GRAPH if lm == A.LOOP_AUTO else A.LOOP_STREAM)
            assert iters_close(st.iters, ref.iters) and st.relres_true <= 2 * s.tol
            for key in ("it_ur32", "it_uz32", "it_uz16"):
                assert switch_close(getattr(st, key), getattr(ref, key), 1)
            # inline scalar steps: no k_epi launches — 4 kernels per iteration + set-up, residual mat-vec (2), finalize
            its = (st.iters + 3) // 4 * 4 if st.loop_mode == A.LOOP_GRAPH else st.iters   # a graph body holds 4 iterations
            assert h.last_launch_count() == 4 * its + 4
        p = torch.rand(s.n, dtype=torch.float64, device="cuda")
        q = g.spmv([p], A.FP64)[0]
        assert np.array_equal(q.cpu().numpy(), O.spmv_fp64(s.rowptr, s.colidx, s.vals, p.cpu().numpy()))
        with pytest.raises(A.AmpPcgError):   # a blob list that does not describe this handle
            bad = A.ShardExport.from_buffer_copy(A.ShardGroup.export(h)); bad.n += 32
            A.ShardGroup.attach_ipc(h, 0, [bytes(bad)])
    finally:
        g.close()


@pytest.mark.parametrize("n", [70, 67, 203])
def test_sharded_halo_wider_than_the_last_rank(n):
    """n not a multiple of 8 and a coupling that reaches the last row: the rounded halo of rank 0 is wider than rank 1's
    row count (n = 70: 6 rows, halo 8), so the push covers rank 1's zero padding.  Two mat-vecs in a row (the second call
    re-uses the pinned state staging while the first one's upload may still be queued), then a solve, then a mat-vec."""
    import types

    sp = pytest.importorskip("scipy.sparse")
    rng = np.random.default_rng(5)
    M = sp.random(n, n, density=0.08, random_state=rng, format="lil")
    for bnd in range(32, n, 32):
        M[bnd - 1, n - 1] = 0.25
        M[bnd, 0] = 0.25
    M = (M + M.T).tocsr()
    M = (M + sp.diags(np.asarray(abs(M).sum(axis=1)).ravel() + 1.0)).tocsr()
    M.sort_indices()
    s = types.SimpleNamespace(n=n, rowptr=M.indptr.astype(np.int32), colidx=M.indices.astype(np.int32),
                              vals=M.data.astype(np.float64), b=rng.uniform(-1, 1, n))
    g, parts = make_group(s, 2)
    try:
        rows1 = parts[1][1] - parts[1][0]
        assert rows1 % 8 != 0 and A.shard_plan(s.rowptr, s.colidx, 2)[0].halo_hi > rows1
        rp, ci, va = (torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals))
        b = torch.from_numpy(s.b).cuda()
        with A.AmpPcg(rp, ci, va) as whole:
            for rep in range(2):
                p64 = torch.from_numpy(rng.uniform(-1, 1, n)).cuda()
                for vec_dt in (torch.float64, torch.float32):
                    p = p64.to(vec_dt)
                    for mat in (A.FP64, A.FP32):
                        q1 = g.spmv(split(p, parts), mat)       # back to back, no synchronisation in between
                        q2 = g.spmv(split(p, parts), mat)
                        assert torch.equal(torch.cat(q1), whole.spmv(p, mat)) and torch.equal(torch.cat(q2), torch.cat(q1))
                spec = POLICY_SPECS["amp_fp64_delay"]
                ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, 1e-10, 500, oracle_policy(spec))
                xs = [torch.zeros(bb - aa, dtype=torch.float64, device="cuda") for aa, bb in parts]
                st = g.solve(split(b, parts), xs, 1e-10, 500, cuda_policy(spec, x0_zero=1))[0]
                assert st.status == ref.status == 0 and abs(st.iters - ref.iters) <= 1, (st.status, st.iters, ref.iters)
                assert st.relres_true <= 2e-10
    finally:
        g.close()
