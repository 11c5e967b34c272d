"""fmm_leaf_multipoles_noalloc (include/fmm.h): the P2M step for all leaves with its scratch in a static device array -- an entry point
that allocates nothing, for callers that cannot reach cudaMalloc.  Checked against the existing path through the C-ABI
(fmm_evaluate_shard_upward for all leaves, then fmm_plan_leaf_multipoles), twice in a row with different charges: the static array
keeps the previous call's contents and the second call must not see them.  Collected last on purpose (the run uses -x)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2511_15269_b200 import fmm, inputs

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-11}  # the north_star tolerance of the parity tests (tests/test_gpu_parity.py)


def rel2(a, b):
    return np.linalg.norm(np.asarray(a, np.float64) - np.asarray(b, np.float64)) / np.linalg.norm(np.asarray(b, np.float64))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def existing_path(P, dq, n_leaves, kp):
    fmm.fmm_evaluate_shard_upward(P.handle, 1, 0, dq)  # permute + P2M of every leaf into the plan's own arrays
    rows = torch.empty((n_leaves, kp), dtype=dq.dtype, device="cuda")
    fmm.fmm_plan_leaf_multipoles(P.handle, 0, 0, n_leaves, rows)
    torch.cuda.synchronize()
    return rows.cpu().numpy()


@pytest.mark.parametrize("dtype,N,N_max,s,p", [(np.float32, 100000, 128, 3, 8), (np.float64, 30000, 32, 2, 6), (np.float32, 5000, 16, 3, 4), (np.float64, 700, 8, 1, 12)])
def test_noalloc_leaf_multipoles_match_the_existing_path_twice_in_a_row(dtype, N, N_max, s, p):
    pos, q1 = inputs.uniform_cube(N, 401, dtype)
    q2 = np.random.default_rng(402).standard_normal(N).astype(dtype)
    P = fmm.Plan(dev(pos), p, N_max, s, 0.77)
    n_leaves, K = P.info["n_leaves"], (p + 1) ** 2
    kp = fmm.fmm_leaf_multipoles_noalloc(P.handle)
    assert kp == fmm.fmm_plan_leaf_multipoles(P.handle, 0, 0, 0) and kp >= K
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    rows = torch.full((n_leaves, kp), float("nan"), dtype=tdt, device="cuda")
    for call, q in enumerate((q1, q2)):  # two calls in a row on the shared static scratch
        dq = dev(q)
        want = existing_path(P, dq, n_leaves, kp)
        rows.fill_(float("nan"))
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        assert fmm.fmm_leaf_multipoles_noalloc(P.handle, dq, rows) == kp
        torch.cuda.synchronize()
        if call == 1:  # (the first call may load kernels lazily) no device memory left the driver's free pool during the call
            assert torch.cuda.mem_get_info()[0] >= free0
        got = rows.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert rel2(got[:, :K], want[:, :K]) <= TOL[dtype], rel2(got[:, :K], want[:, :K])
        assert np.all(got[:, K:] == 0)  # the padding of a row is defined
    # the plan was not written: its forward evaluate still answers for the charges of ITS last upward pass, and a fresh evaluate works
    u, f = P.evaluate(dev(q1))
    assert bool(torch.isfinite(u).all()) and bool(torch.isfinite(f).all())
    P.close()


def test_noalloc_rejects_sizes_beyond_the_static_array():
    n_max = fmm.FMM_NOALLOC_MAX_BYTES // 16
    N = n_max + 1
    pos, q = inputs.uniform_cube(N, 403, np.float32)
    P = fmm.Plan(dev(pos), 2, 128, 3, 0.77)
    kp = fmm.fmm_leaf_multipoles_noalloc(P.handle)  # the query works at any size
    rows = torch.full((P.info["n_leaves"], kp), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(fmm.FmmError) as e:
        fmm.fmm_leaf_multipoles_noalloc(P.handle, dev(q), rows)
    assert "FMM_NOALLOC_MAX_BYTES" in str(e.value) and str(N) in str(e.value)
    torch.cuda.synchronize()
    assert bool((rows == 7.0).all())  # nothing was launched
    P.close()
    # exactly at the limit it runs
    pos, q = inputs.uniform_cube(n_max, 404, np.float32)
    P = fmm.Plan(dev(pos), 2, 128, 3, 0.77)
    rows = torch.empty((P.info["n_leaves"], kp), dtype=torch.float32, device="cuda")
    dq = dev(q)
    fmm.fmm_leaf_multipoles_noalloc(P.handle, dq, rows)
    want = existing_path(P, dq, P.info["n_leaves"], kp)
    assert rel2(rows.cpu().numpy()[:, :9], want[:, :9]) <= 1e-5
    # separate-target plans are refused
    PT = fmm.PlanTargets(dev(pos[:1000]), dev(pos[1000:3000]), 2, 32, 2)
    with pytest.raises(fmm.FmmError):
        fmm.fmm_leaf_multipoles_noalloc(PT.handle, dq[:1000].contiguous(), rows)
    PT.close()
    P.close()
