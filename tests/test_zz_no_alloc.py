"""-m gpu: amp_xr_update_static, the one entry point of the library that allocates nothing, against the handle path.

Why it exists: some users of this library can't let it call cudaMalloc.  A process that handed the whole device memory
to its own pool at start-up gets out-of-memory from any later cudaMalloc, and a loop with a latency bound can't take the
device-wide synchronisation an allocation may cost.  Every other entry point needs a handle, whose create() allocates;
amp_xr_update_static runs step a5 (x += alpha p, r -= alpha q, delta = ||r||; Alg 4.1 lines 15-17) on
the caller's own arrays and keeps the scratch memory of its grid reduction in a static device array inside the library
(131 328 bytes per GPU, which limits it to XR_STATIC_MAX_N = 67 108 864 elements).

What is checked: on the same inputs, x and r are bit-identical to what the existing path (k_xr through
amp_pcg_debug_step, FP64 phase) leaves, and delta agrees to n 2^-53 relative (two fixed but different summation orders,
the tolerance of tests/test_gpu_steps.py) — on TWO calls in a row, the second on a smaller odd n, because all calls share
the one scratch array and it keeps the first call's partial sums and ticket.  The first call made in a process also does
the per-device set-up (address look-up of the array), so the file passes alone in a fresh process as well as after the
rest of the suite.  It is named test_zz_* so that pytest collects it last: with -x a failure here hides no other test.
"""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")


def _existing_path(s, alpha, p, q, x, r):
    """x, r, delta after one FP64 x / r update through the handle's own kernel (k_xr)."""
    with A.AmpPcg(*(torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals)), A.PRECOND_JACOBI,
                  vec_kernel=A.VEC_DIRECT) as h:
        h.debug_set_vector(A.VEC_P, torch.from_numpy(p).cuda())
        h.debug_set_vector(A.VEC_Q, torch.from_numpy(q).cuda())
        h.debug_set_vector(A.VEC_R, torch.from_numpy(r).cuda())
        xd = torch.from_numpy(x).cuda()
        io = h.debug_step(A.STEP_XR, x=xd, rs=A.FP64, ur=A.FP64, uz=A.FP64, ps=A.FP64, ur_n=A.FP64, uz_n=A.FP64, alpha=alpha)
        return xd.cpu().numpy(), h.debug_get_vector(A.VEC_R, A.FP64).cpu().numpy(), io.sum0


def _same_bits(got, want):
    return np.array_equal(got.view(np.uint64), want.view(np.uint64))


def test_no_alloc_xr_update_matches_handle_path_twice_in_a_row():
    # first call: 103 823 elements = 26 tiles of 4096 with a ragged, odd tail; second call: 1331 elements = one tile,
    # launched over the scratch contents the first call left behind
    calls = []
    for (name, size, alpha, seed) in (("c2", 47, 0.731, 11), ("c3", 11, -2.5e-3, 12)):
        s = make_config(name, size)
        assert s.n % 2 == 1
        rng = np.random.default_rng(seed)
        p, q, x, r = (rng.standard_normal(s.n) for _ in range(4))
        r[:4] = (0.0, -0.0, 1e-300, 1e150)
        calls.append((s, alpha, p, q, x, r, _existing_path(s, alpha, p, q, x, r)))
    torch.cuda.synchronize()
    results = []
    for s, alpha, p, q, x, r, _ in calls:  # back to back on one stream, nothing in between
        pd, qd, xd, rd = (torch.from_numpy(a).cuda() for a in (p, q, x, r))
        delta = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
        A.xr_update_static(alpha, pd, qd, xd, rd, delta)
        results.append((pd, qd, xd, rd, delta))
    torch.cuda.synchronize()
    for (s, alpha, p, q, x, r, (x_ref, r_ref, delta_ref)), (pd, qd, xd, rd, delta) in zip(calls, results):
        assert _same_bits(xd.cpu().numpy(), x_ref), "x"
        assert _same_bits(rd.cpu().numpy(), r_ref), "r"
        assert _same_bits(pd.cpu().numpy(), p) and _same_bits(qd.cpu().numpy(), q), "p, q are read-only"
        assert float(delta[0]) == pytest.approx(delta_ref, rel=s.n * 2.0 ** -53)
        assert float(delta[0]) == pytest.approx(float(np.sqrt(np.sum(r_ref.astype(np.longdouble) ** 2))), rel=s.n * 2.0 ** -53)


def test_no_alloc_xr_update_rejects_what_the_static_array_cannot_serve():
    t = torch.zeros(8, dtype=torch.float64, device="cuda")
    d = torch.zeros(1, dtype=torch.float64, device="cuda")
    L = A.load_library()
    ptr = t.data_ptr()
    for n in (A.XR_STATIC_MAX_N + 1, 0, -5):
        assert L.amp_xr_update_static(n, 1.0, ptr, ptr, ptr, ptr, d.data_ptr(), None) == -1
    assert L.amp_xr_update_static(A.XR_STATIC_MAX_N + 1, 1.0, ptr, ptr, ptr, ptr, d.data_ptr(), None) == -1
    assert "AMP_XR_STATIC_MAX_N" in L.amp_pcg_last_error().decode()
    assert L.amp_xr_update_static(8, 1.0, ptr + 8, ptr, ptr, ptr, d.data_ptr(), None) == -1  # misaligned p
    assert L.amp_xr_update_static(8, 1.0, None, ptr, ptr, ptr, d.data_ptr(), None) == -1
    torch.cuda.synchronize()
    assert float(t.abs().sum()) == 0.0 and float(d[0]) == 0.0  # nothing ran
