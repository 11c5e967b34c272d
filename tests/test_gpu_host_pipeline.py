"""The host path as a two-deep pipeline (include/fmm.h fmm_evaluate_host_submit / fmm_evaluate_host_wait): the copies of one call run
beside the kernels of the next.  Every call must deliver exactly what the synchronous fmm_evaluate_host delivers (north_star
tolerance against the oracle), in submission order, with different charges in flight at the same time; the depth limit and
the empty wait are status codes."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-11}


def rel2(a, b):
    return np.linalg.norm(np.asarray(a, np.float64) - b) / np.linalg.norm(b)


def pinned(shape, tdt):
    return torch.empty(shape, dtype=tdt).pin_memory()


@pytest.mark.parametrize("dtype,N,N_max,s,p", [(np.float32, 30000, 32, 3, 8), (np.float64, 5000, 64, 3, 6), (np.float32, 300000, 128, 3, 4)])
def test_pipelined_calls_match_the_oracle_in_order(dtype, N, N_max, s, p):
    pos, q0 = inputs.uniform_cube(N, 411, dtype)
    f32 = dtype == np.float32
    tdt = torch.float32 if f32 else torch.float64
    P = fmm.Plan(torch.from_numpy(pos).cuda(), p, N_max, s, 0.77)
    Po = O.Plan(pos, p, N_max, s, 0.77)
    n_calls = 5
    qs = [(q0 * (1.0 + 0.5 * k) - 0.1 * k).astype(dtype) for k in range(n_calls)]  # a different charge vector per call
    want = [Po.evaluate(qk, fp32_rule=f32) for qk in qs]
    hq = [torch.from_numpy(qk).pin_memory() for qk in qs]
    outs = [(pinned(N, tdt), pinned((N, 3), tdt)) for _ in range(2)]
    got = []
    for k in range(n_calls):
        if k >= 2:
            fmm.fmm_evaluate_host_wait(P.handle)           # call k-2 has delivered: its buffers are ours again
            u, f = outs[k & 1]
            got.append((u.numpy().copy(), f.numpy().copy()))
        u, f = outs[k & 1]
        u.fill_(float("nan")); f.fill_(float("nan"))
        fmm.fmm_evaluate_host_submit(P.handle, hq[k], u, f)
    for k in range(n_calls - 2, n_calls):
        fmm.fmm_evaluate_host_wait(P.handle)
        u, f = outs[k & 1]
        got.append((u.numpy().copy(), f.numpy().copy()))
    for k in range(n_calls):
        assert rel2(got[k][0], want[k][0]) <= TOL[dtype] and rel2(got[k][1], want[k][1]) <= TOL[dtype], k
    # the synchronous call still works after the pipeline has drained, potential only
    hu = pinned(N, tdt)
    fmm.fmm_evaluate_host(P.handle, hq[1], hu, None)
    assert rel2(hu.numpy(), want[1][0]) <= TOL[dtype]
    P.close()


def test_depth_limit_and_empty_wait_are_status_codes():
    N = 2000
    pos, q = inputs.uniform_cube(N, 412, np.float32)
    P = fmm.Plan(torch.from_numpy(pos).cuda(), 4, 32, 2, 0.77)
    with pytest.raises(fmm.FmmError) as e:
        fmm.fmm_evaluate_host_wait(P.handle)
    assert e.value.status == fmm.FMM_ERR_INVALID_ARG
    hq = torch.from_numpy(q).pin_memory()
    bufs = [(pinned(N, torch.float32), pinned((N, 3), torch.float32)) for _ in range(3)]
    fmm.fmm_evaluate_host_submit(P.handle, hq, *bufs[0])
    fmm.fmm_evaluate_host_submit(P.handle, hq, *bufs[1])
    with pytest.raises(fmm.FmmError) as e:
        fmm.fmm_evaluate_host_submit(P.handle, hq, *bufs[2])
    assert e.value.status == fmm.FMM_ERR_UNSUPPORTED and "in flight" in str(e.value)
    fmm.fmm_evaluate_host_wait(P.handle)
    fmm.fmm_evaluate_host_wait(P.handle)
    assert torch.equal(bufs[0][0], bufs[1][0]) or rel2(bufs[0][0].numpy(), bufs[1][0].numpy().astype(np.float64)) <= 2e-6  # same charges: same result up to the atomics
    # separate targets: charges live on the sources, outputs on the targets
    tp = np.ascontiguousarray((np.random.default_rng(5).random((1500, 3)) * 1.2 - 0.1).astype(np.float32))
    Pt = fmm.PlanTargets(torch.from_numpy(pos).cuda(), torch.from_numpy(tp).cuda(), 6, 32, 2, 0.77)
    uo, fo = O.PlanST(pos, tp, 6, 32, 2, 0.77).evaluate(q, fp32_rule=True)
    hu, hf = pinned(1500, torch.float32), pinned((1500, 3), torch.float32)
    fmm.fmm_evaluate_host_submit(Pt.handle, hq, hu, hf)
    fmm.fmm_evaluate_host_wait(Pt.handle)
    assert rel2(hu.numpy(), uo) <= 1e-5 and rel2(hf.numpy(), fo) <= 1e-5
    Pt.close()
    P.close()
