"""CUDA-graph replay of the evaluate schedule (include/fmm.h fmm_plan_set_graph): repeated evaluates with the same device pointers
run as one cudaGraphLaunch.  The graph holds the same kernels on the same data, so every replay must meet the north_star tolerance
against the oracle, survive a re-plan (the graph is dropped), alternate with adjoint evaluates, and the evaluate must still be
capturable into a graph of the caller."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-11}


def rel2(a, b):
    return np.linalg.norm(np.asarray(a, np.float64) - b) / np.linalg.norm(b)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s,p,cross,serial", [(4096, 128, 3, 6, 0, 0), (20000, 16, 3, 8, 0, 0), (20000, 16, 3, 8, 1, 0), (3000, 32, 2, 10, 0, 1), (700, 4, 1, 4, 1, 0)])
def test_graph_replays_match_the_oracle(dtype, N, N_max, s, p, cross, serial):
    pos, q = inputs.uniform_cube(N, 301, dtype)
    P = fmm.Plan(dev(pos), p, N_max, s, 0.77, cross_level=cross)
    fmm.fmm_plan_set_schedule(P.handle, serial)
    Po = O.Plan(pos, p, N_max, s, 0.77, cross_level=cross)
    f32 = dtype == np.float32
    dq = dev(q)
    tdt = torch.float32 if f32 else torch.float64
    u, f = torch.empty(N, dtype=tdt, device="cuda"), torch.empty((N, 3), dtype=tdt, device="cuda")
    uo, fo = Po.evaluate(q, fp32_rule=f32)
    for rep in range(5):  # 1: plain, 2: capture + launch, 3..: replays
        u.fill_(float("nan")); f.fill_(float("nan"))
        fmm.fmm_evaluate(P.handle, dq, u, f)
        assert rel2(u.cpu().numpy(), uo) <= TOL[dtype] and rel2(f.cpu().numpy(), fo) <= TOL[dtype], rep
    # new charges in the SAME buffer: the replay reads them
    q2 = (q * 0.5 + 0.25).astype(dtype)
    dq.copy_(dev(q2))
    uo2, fo2 = Po.evaluate(q2, fp32_rule=f32)
    fmm.fmm_evaluate(P.handle, dq, u, f)
    assert rel2(u.cpu().numpy(), uo2) <= TOL[dtype] and rel2(f.cpu().numpy(), fo2) <= TOL[dtype]
    # potential only: another pointer set, another graph
    for rep in range(3):
        u.fill_(float("nan"))
        fmm.fmm_evaluate(P.handle, dq, u, None)
        assert rel2(u.cpu().numpy(), uo2) <= TOL[dtype]
    # graphs off: plain launches, same answer
    fmm.fmm_plan_set_graph(P.handle, 0)
    fmm.fmm_evaluate(P.handle, dq, u, f)
    assert rel2(u.cpu().numpy(), uo2) <= TOL[dtype] and rel2(f.cpu().numpy(), fo2) <= TOL[dtype]
    P.close()


def test_graph_is_dropped_by_a_replan_and_by_the_schedule_switches():
    N, p = 6000, 6
    pos, q = inputs.uniform_cube(N, 302, np.float64)
    P = fmm.Plan(dev(pos), p, 32, 3, 0.77)
    dq = dev(q)
    u, f = torch.empty(N, dtype=torch.float64, device="cuda"), torch.empty((N, 3), dtype=torch.float64, device="cuda")
    for _ in range(3):
        fmm.fmm_evaluate(P.handle, dq, u, f)
    pos2 = np.ascontiguousarray(np.random.default_rng(303).random((N, 3)) ** 2)  # a different tree and different lists
    P.update(dev(pos2))
    uo, fo = O.Plan(pos2, p, 32, 3, 0.77).evaluate(q)
    for _ in range(3):
        fmm.fmm_evaluate(P.handle, dq, u, f)
        assert rel2(u.cpu().numpy(), uo) <= 1e-11 and rel2(f.cpu().numpy(), fo) <= 1e-11
    for variant, det in ((1, 0), (0, 1), (0, 0)):
        fmm.fmm_plan_set_m2l_variant(P.handle, variant)
        fmm.fmm_plan_set_deterministic(P.handle, det)
        got = []
        for _ in range(3):
            fmm.fmm_evaluate(P.handle, dq, u, f)
            assert rel2(u.cpu().numpy(), uo) <= 1e-11 and rel2(f.cpu().numpy(), fo) <= 1e-11
            got.append(u.cpu().numpy().copy())
        if det:
            assert np.array_equal(got[0], got[1]) and np.array_equal(got[1], got[2])  # plain run and replays: identical bits
    P.close()


@pytest.mark.parametrize("cross", [0, 1])
def test_forward_and_adjoint_alternate(cross):
    """an optimisation loop calls evaluate and evaluate_adjoint in turn with the same buffers: both are replayed from the cache"""
    N, p = 2500, 6
    pos, q = inputs.uniform_cube(N, 304, np.float64)
    rng = np.random.default_rng(305)
    ubar = rng.standard_normal(N)
    P = fmm.Plan(dev(pos), p, 32, 2, 0.77, cross_level=cross)
    Po = O.Plan(pos, p, 32, 2, 0.77, cross_level=cross)
    uo, _ = Po.evaluate(q)
    go = Po.evaluate_adjoint(ubar, None)
    dq, dub = dev(q), dev(ubar)
    u, g = torch.empty(N, dtype=torch.float64, device="cuda"), torch.empty(N, dtype=torch.float64, device="cuda")
    for _ in range(4):
        u.fill_(float("nan")); g.fill_(float("nan"))
        fmm.fmm_evaluate(P.handle, dq, u, None)
        fmm.fmm_evaluate_adjoint(P.handle, dub, None, g)
        assert rel2(u.cpu().numpy(), uo) <= 1e-11
        assert rel2(g.cpu().numpy(), go) <= 1e-11
    P.close()


def test_separate_targets_and_host_buffers():
    sp, q = inputs.uniform_cube(3000, 306, np.float32)
    tp = (np.random.default_rng(307).random((5000, 3)) * 1.4 - 0.2).astype(np.float32)
    P = fmm.PlanTargets(dev(sp), dev(tp), 8, 32, 2)
    uo, fo = O.PlanST(sp, tp, 8, 32, 2).evaluate(q, fp32_rule=True)
    dq = dev(q)
    u, f = torch.empty(5000, dtype=torch.float32, device="cuda"), torch.empty((5000, 3), dtype=torch.float32, device="cuda")
    for _ in range(4):
        u.fill_(float("nan")); f.fill_(float("nan"))
        fmm.fmm_evaluate(P.handle, dq, u, f)
        assert rel2(u.cpu().numpy(), uo) <= 1e-5 and rel2(f.cpu().numpy(), fo) <= 1e-5
    P.close()
    pos, q = inputs.uniform_cube(5000, 308, np.float32)
    P = fmm.Plan(dev(pos), 8, 64, 3, 0.77)
    uo, fo = O.Plan(pos, 8, 64, 3, 0.77).evaluate(q, fp32_rule=True)
    hq = torch.from_numpy(q).pin_memory()
    hu, hf = torch.empty(5000, dtype=torch.float32).pin_memory(), torch.empty((5000, 3), dtype=torch.float32).pin_memory()
    for _ in range(4):
        hu.fill_(float("nan")); hf.fill_(float("nan"))
        fmm.fmm_evaluate_host(P.handle, hq, hu, hf)
        torch.cuda.synchronize()
        assert rel2(hu.numpy(), uo) <= 1e-5 and rel2(hf.numpy(), fo) <= 1e-5
    P.close()


def test_the_caller_can_capture_an_evaluate_into_their_own_graph():
    N, p = 5000, 6
    pos, q = inputs.uniform_cube(N, 309, np.float64)
    P = fmm.Plan(dev(pos), p, 64, 3, 0.77)
    uo, fo = O.Plan(pos, p, 64, 3, 0.77).evaluate(q)
    dq = dev(q)
    u, f = torch.empty(N, dtype=torch.float64, device="cuda"), torch.empty((N, 3), dtype=torch.float64, device="cuda")
    fmm.fmm_evaluate(P.handle, dq, u, f)  # one-time work (function attributes, constant upload) happens outside the capture
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    G = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        G.capture_begin()
        fmm.fmm_evaluate(P.handle, dq, u, f, stream=side)
        y = u * 2.0  # the caller's own work behind the evaluate, in the same graph
        G.capture_end()
    torch.cuda.synchronize()
    for _ in range(3):
        u.fill_(float("nan")); f.fill_(float("nan"))
        G.replay()
        torch.cuda.synchronize()
        assert rel2(u.cpu().numpy(), uo) <= 1e-11 and rel2(f.cpu().numpy(), fo) <= 1e-11
        assert rel2(y.cpu().numpy(), 2.0 * uo) <= 1e-11
    P.close()


def test_the_binding_rejects_tensors_that_do_not_fit_the_plan():
    """the C side sees raw pointers only: dtype, shape, contiguity and residency are checked where the tensors still exist"""
    pos, q = inputs.uniform_cube(1000, 310, np.float32)
    P = fmm.Plan(dev(pos), 4, 32, 2, 0.77)
    dq = dev(q)
    u, f = torch.empty(1000, dtype=torch.float32, device="cuda"), torch.empty((1000, 3), dtype=torch.float32, device="cuda")
    fmm.fmm_evaluate(P.handle, dq, u, f)
    for bad in (dict(charges=dq.double()), dict(charges=dq[:999]), dict(charges=dq.cpu()), dict(potential=u.double()), dict(field=f.t().contiguous()),
                dict(field=torch.empty((1000, 6), dtype=torch.float32, device="cuda")[:, ::2]), dict(charges=q)):
        args = dict(charges=dq, potential=u, field=f)
        args.update(bad)
        with pytest.raises(ValueError):
            fmm.fmm_evaluate(P.handle, args["charges"], args["potential"], args["field"])
    with pytest.raises(ValueError):
        fmm.fmm_evaluate_host(P.handle, dq, u.cpu(), f.cpu())  # the host path wants host buffers
    h = P.handle
    P.close()
    with pytest.raises(ValueError):
        fmm.fmm_evaluate(h, dq, u, f)  # a destroyed handle never reaches the library
