"""fmm_plan_update (first half): re-planning an existing plan for moved points must give
exactly the plan a fresh fmm_plan_create gives -- hierarchy and lists bit-exact against a fresh ORACLE plan of the new positions --
and evaluates (forward and adjoint) on the updated plan must meet the parity tolerance."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs
from test_gpu_parity import TOL, assert_same_hierarchy, rel2

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s,p,cross", [(20000, 32, 3, 6, 0), (5000, 16, 2, 5, 1), (3000, 8, 1, 4, 0), (129, 128, 3, 3, 0)])
def test_update_equals_fresh_plan(dtype, N, N_max, s, p, cross):
    pos, q = inputs.uniform_cube(N, 201, dtype)
    P = fmm.Plan(dev(pos), p, N_max, s, 0.77, cross_level=cross)
    P.evaluate(dev(q))
    if cross:
        P.evaluate_adjoint(dev(q), None)  # builds the adjoint view of the OLD positions: must be dropped by the update
    rng = np.random.default_rng(202)
    for step, amp in enumerate((0.01, 0.3)):  # a 1 % jiggle, then a displacement that reshuffles the tree
        pos = (pos.astype(np.float64) + amp * rng.standard_normal(pos.shape) * (1.0 / N) ** (1 / 3)).astype(dtype)
        P.update(dev(pos))
        Po = O.Plan(pos, p, N_max, s, 0.77, cross_level=cross)
        assert_same_hierarchy(P, Po, dtype)
        u, f = P.evaluate(dev(q))
        torch.cuda.synchronize()
        uo, fo = Po.evaluate(q, fp32_rule=dtype == np.float32)
        assert rel2(u.cpu().numpy(), uo) <= TOL[dtype] and rel2(f.cpu().numpy(), fo) <= TOL[dtype], (step, amp)
        if N <= 5000:
            g = P.evaluate_adjoint(dev(q), None).cpu().numpy()
            assert rel2(g, Po.evaluate_adjoint(q, None, fp32_rule=dtype == np.float32)) <= TOL[dtype]
    P.close()


def test_update_separate_targets_and_errors():
    sp, q = inputs.uniform_cube(4000, 203, np.float32)
    tp = (np.random.default_rng(204).random((3000, 3)) * 1.4 - 0.2).astype(np.float32)
    P = fmm.PlanTargets(dev(sp), dev(tp), 6, 32, 2)
    tp2 = (tp + np.float32(0.02) * np.random.default_rng(205).standard_normal(tp.shape).astype(np.float32))
    P.update(targets=dev(tp2))  # only the targets moved: the source hierarchy is kept
    Po = O.PlanST(sp, tp2, 6, 32, 2)
    lg, lo_ = P.lists(), Po.lists()
    for k in ("weak_off", "weak_src", "strong_off", "strong_src"):
        assert np.array_equal(lg[k].astype(np.int64), lo_[k]), k
    assert lg["steps"].tolist() == lo_["steps"].tolist()
    u, f = P.evaluate(dev(q))
    uo, fo = Po.evaluate(q, fp32_rule=True)
    assert rel2(u.cpu().numpy(), uo) <= 1e-5 and rel2(f.cpu().numpy(), fo) <= 1e-5
    sp2 = (sp + np.float32(0.01) * np.random.default_rng(206).standard_normal(sp.shape).astype(np.float32))
    P.update(sources=dev(sp2), targets=dev(tp))
    Po = O.PlanST(sp2, tp, 6, 32, 2)
    u, f = P.evaluate(dev(q))
    uo, fo = Po.evaluate(q, fp32_rule=True)
    assert rel2(u.cpu().numpy(), uo) <= 1e-5 and rel2(f.cpu().numpy(), fo) <= 1e-5
    with pytest.raises(ValueError):
        P.update(sources=dev(sp2[:100]))
    with pytest.raises(fmm.FmmError):
        fmm.fmm_plan_update(P.handle, None, None)
    P.close()


def test_update_one_million_timing():
    """N = 1M (config 2): a 1 % displacement step; bit-exact lists against the oracle, and the device time of the update is printed"""
    pos, q, c = inputs.make("cfg2_cube1M_f32")
    P = fmm.Plan(dev(pos), c["p"], c["N_max"], c["s"], c["theta"])
    rng = np.random.default_rng(207)
    ms = []
    for _ in range(3):
        pos = (pos + np.float32(1e-4) * rng.standard_normal(pos.shape).astype(np.float32))
        d = dev(pos)
        P.update(d)
        ms.append(P.timings())
    Po = O.Plan(pos, c["p"], c["N_max"], c["s"], c["theta"])
    assert_same_hierarchy(P, Po, np.float32)
    print("fmm_plan_update at N = 1M, device ms:", ms)
    P.close()
