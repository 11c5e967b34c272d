"""GPU parity for separate sources and targets (fmm_plan_create_targets): both hierarchies, the level march and
both lists bit-exact against the oracle; potential and field at the targets within the north_star tolerances; error against
the plain definition within 1.5x the oracle's own."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-11}


def rel2(a, b):
    return np.linalg.norm(np.asarray(a, np.float64) - b) / np.linalg.norm(b)


def targets(n, seed, dtype, lo=-0.3, hi=1.4):
    t = np.random.default_rng(seed).random((n, 3)) * (hi - lo) + lo
    return np.ascontiguousarray(t.astype(dtype))


def same_tree(tg, to):
    assert np.array_equal(tg["perm"].astype(np.int64), to["perm"])
    assert np.array_equal(tg["box_count"].astype(np.int64), to["box_count"])
    ne = to["box_count"] > 0
    assert np.array_equal(tg["box_start"].astype(np.int64)[ne], to["box_start"][ne])
    assert np.array_equal(tg["lo"].astype(np.float64)[ne], to["lo"][ne]) and np.array_equal(tg["hi"].astype(np.float64)[ne], to["hi"][ne])
    assert np.array_equal(tg["ctr"][ne], to["ctr"][ne]) and np.array_equal(tg["rad"][ne], to["rad"][ne])


def run_st(sp, q, tp, p, N_max, s, theta=0.77, direct=True, variants=(0,)):
    dt = sp.dtype.type
    P = fmm.PlanTargets(torch.from_numpy(sp).cuda(), torch.from_numpy(tp).cuda(), p, N_max, s, theta)
    Po = O.PlanST(sp, tp, p, N_max, s, theta)
    assert (P.info["L"], P.info["n_boxes"], P.info["n_leaves"]) == (Po.info["tgt"]["L"], Po.info["tgt"]["n_boxes"], Po.info["tgt"]["n_leaves"])
    assert (P.source_info["L"], P.source_info["n_boxes"], P.source_info["N"]) == (Po.info["src"]["L"], Po.info["src"]["n_boxes"], sp.shape[0])
    same_tree(P.tree("tgt"), Po.tree("tgt"))
    same_tree(P.tree("src"), Po.tree("src"))
    lg, lo_ = P.lists(), Po.lists()
    assert lg["steps"].tolist() == lo_["steps"].tolist()
    assert (P.info["n_weak"], P.info["n_strong"], P.info["n_p2p_pairs"]) == (Po.n_weak, Po.n_strong, Po.n_p2p_pairs)
    for k in ("weak_off", "weak_src", "strong_off", "strong_src"):
        assert np.array_equal(lg[k].astype(np.int64), lo_[k]), k
    f32 = dt == np.float32
    uo, fo = Po.evaluate(q, fp32_rule=f32)
    tq = torch.from_numpy(np.ascontiguousarray(q)).cuda()
    res = None
    for v in variants:
        fmm.fmm_plan_set_m2l_variant(P.handle, v)
        for serial in (0, 1):
            fmm.fmm_plan_set_schedule(P.handle, serial)
            u, f = P.evaluate(tq)
            torch.cuda.synchronize()
            u, f = u.cpu().numpy(), f.cpu().numpy()
            assert np.all(np.isfinite(u)) and np.all(np.isfinite(f))
            eu, ef = rel2(u, uo), rel2(f, fo)
            assert eu <= TOL[dt] and ef <= TOL[dt], (v, serial, eu, ef)
            res = (u, f)
    if direct:
        ud, fd = O.direct_st(sp, q, tp, fp32_rule=f32)
        # north_star: GPU error <= 1.5 x the oracle's own.  The slack is the unit roundoff of the plan's dtype times 8 -- where the oracle is
        # exact to fp64 rounding (all-P2P cases) an fp32 result can only be as close to the definition as binary32 arithmetic allows;
        # it never dominates a truncation error (>= 1e-6 in every far-field case here), so the 1.5x clause keeps its meaning
        slack = 8 * (6e-8 if f32 else 1.2e-16)
        assert rel2(res[0], ud) <= 1.5 * rel2(uo, ud) + slack and rel2(res[1], fd) <= 1.5 * rel2(fo, fd) + slack
    st = fmm.fmm_evaluate_profiled(P.handle, tq, *P.evaluate(tq))
    assert st["total"] > 0
    P.close()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("Ns,Nt,N_max,s,p", [(3000, 2000, 32, 2, 6), (1024, 4096, 16, 3, 8), (5000, 700, 20, 1, 4), (2500, 2500, 8, 3, 10)])
def test_separate_targets(dtype, Ns, Nt, N_max, s, p):
    sp, q = inputs.uniform_cube(Ns, 61, dtype)
    run_st(sp, q, targets(Nt, 62, dtype), p, N_max, s)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_separate_targets_generic_kernels_agree(dtype):
    """m2l_variant 1 (generic warp-per-box kernels, generic P2P) is an independent implementation of the same path."""
    sp, q = inputs.uniform_cube(2000, 63, dtype)
    run_st(sp, q, targets(1500, 64, dtype), 5, 16, 2, variants=(0, 1))


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_identical_sets_equal_the_cross_level_plan(dtype):
    """Sources == targets: lists equal those of fmm_plan_create with cross_level = 1; self pairs drop out by zero distance (S3)."""
    pos, q = inputs.uniform_cube(3000, 65, dtype)
    run_st(pos, q, pos.copy(), 6, 32, 2, direct=False)
    tp = torch.from_numpy(pos).cuda()
    P1 = fmm.Plan(tp, 6, 32, 2, 0.77, cross_level=1)
    P2 = fmm.PlanTargets(tp, tp.clone(), 6, 32, 2, 0.77)
    l1, l2 = P1.lists(), P2.lists()
    for k in ("weak_off", "weak_src", "strong_off", "strong_src"):
        assert np.array_equal(l1[k], l2[k])
    P1.close()
    P2.close()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_degenerate_geometries(dtype):
    sp, q = inputs.uniform_cube(500, 66, dtype)
    # far-away targets: the march ends without strong pairs (empty P2P lists for every target leaf)
    run_st(sp, q, targets(300, 67, dtype, 20.0, 21.0), 8, 16, 2)
    # a single target / a single source / fewer points than one leaf holds
    run_st(sp, q, targets(1, 68, dtype), 6, 16, 2)
    run_st(sp[:1].copy(), q[:1].copy(), targets(400, 69, dtype), 6, 16, 2)
    run_st(sp[:10].copy(), q[:10].copy(), targets(7, 70, dtype), 6, 16, 2)
    # targets on a plane inside the source cloud (degenerate target boxes), a few coinciding with sources
    tp = targets(900, 71, dtype, 0.0, 1.0)
    tp[:, 2] = dtype(0.5)
    tp[:50] = sp[:50]
    run_st(sp, q, np.ascontiguousarray(tp), 6, 16, 2)


def test_shield_demo_shape():
    """The geometry of PAPER.md:281-300: 128 + 256 charges on spheres of radius 2 and 5, 1024 + 1024 sample points on spheres of radius 1.5 and 2.5."""
    rng = np.random.default_rng(72)
    def sphere(n, r):
        v = rng.normal(size=(n, 3))
        return r * v / np.linalg.norm(v, axis=1, keepdims=True)
    sp = np.ascontiguousarray(np.concatenate([sphere(128, 2.0), sphere(256, 5.0)]))
    q = rng.uniform(-1, 1, sp.shape[0])
    tp = np.ascontiguousarray(np.concatenate([sphere(1024, 1.5), sphere(1024, 2.5)]))
    run_st(sp, q, tp, 8, 32, 2)


def test_host_path_and_partial_outputs():
    sp, q = inputs.uniform_cube(4000, 73, np.float32)
    tp = targets(3000, 74, np.float32)
    P = fmm.PlanTargets(torch.from_numpy(sp).cuda(), torch.from_numpy(tp).cuda(), 6, 32, 3)
    tq = torch.from_numpy(q).cuda()
    u, f = P.evaluate(tq)
    u2, _ = P.evaluate(tq, want_field=False)
    _, f2 = P.evaluate(tq, want_potential=False)
    torch.cuda.synchronize()
    assert rel2(u2.cpu().numpy(), u.double().cpu().numpy()) < 1e-6 and rel2(f2.cpu().numpy(), f.double().cpu().numpy()) < 1e-6
    hu, hf = np.empty(3000, np.float32), np.empty((3000, 3), np.float32)
    fmm.fmm_evaluate_host(P.handle, q, hu, hf)
    assert rel2(hu, u.double().cpu().numpy()) < 1e-6 and rel2(hf, f.double().cpu().numpy()) < 1e-6
    P.close()


def test_one_million_sources_sampled_targets():
    """Config-2 sources (N = 1M, fp32, p = 8) evaluated at 200 000 separate targets: both hierarchies, the march and both lists
    bit-exact against the oracle at full size; potential / field on the targets of 128 random target leaves against the oracle
    (leaf mask: same arithmetic as a full run) at the north_star tolerance and element by element, and against the definition."""
    sp, q, c = inputs.make("cfg2_cube1M_f32")
    tp = targets(200000, 75, np.float32, 0.0, 1.0)
    P = fmm.PlanTargets(torch.from_numpy(sp).cuda(), torch.from_numpy(tp).cuda(), c["p"], c["N_max"], c["s"], c["theta"])
    Po = O.PlanST(sp, tp, c["p"], c["N_max"], c["s"], c["theta"])
    same_tree(P.tree("tgt"), Po.tree("tgt"))
    same_tree(P.tree("src"), Po.tree("src"))
    lg, lo_ = P.lists(), Po.lists()
    assert lg["steps"].tolist() == lo_["steps"].tolist()
    assert (P.info["n_weak"], P.info["n_strong"], P.info["n_p2p_pairs"]) == (Po.n_weak, Po.n_strong, Po.n_p2p_pairs)
    for k in ("weak_off", "weak_src", "strong_off", "strong_src"):
        assert np.array_equal(lg[k].astype(np.int64), lo_[k]), k
    u, f = P.evaluate(torch.from_numpy(q).cuda())
    torch.cuda.synchronize()
    u, f = u.cpu().numpy(), f.cpu().numpy()
    nl = Po.info["tgt"]["n_leaves"]
    mask = np.zeros(nl, np.uint8)
    mask[np.random.default_rng(0).choice(nl, 128, replace=False)] = 1
    uo, fo = Po.evaluate(q, leaf_mask=mask, fp32_rule=True)
    sel = np.flatnonzero(np.isfinite(uo))
    assert sel.size > 1000
    eu, ef = rel2(u[sel], uo[sel]), rel2(f[sel], fo[sel])
    assert eu <= 1e-5 and ef <= 1e-5, (eu, ef)
    assert np.max(np.abs(u[sel] - uo[sel])) <= 1e-4 * np.max(np.abs(uo[sel])) and np.max(np.abs(f[sel] - fo[sel])) <= 1e-4 * np.max(np.abs(fo[sel]))
    dsel = sel[:1024]
    ud, fd = O.direct_st(sp, q, tp[dsel], fp32_rule=True)
    assert rel2(u[dsel], ud) <= 1.5 * rel2(uo[dsel], ud) and rel2(f[dsel], fd) <= 1.5 * rel2(fo[dsel], fd)
    P.close()
