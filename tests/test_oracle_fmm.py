"""Whole-oracle pins: FMM vs the plain O(N^2) definition (eqs. 1-3), error decay with p (eq. 5),
permutation invariance, masked == full evaluation, linearity in q, and the accuracy order the paper reports."""
import numpy as np
import pytest

from oracle import api as O
from paper_2511_15269_b200 import inputs


def rel2(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def test_direct_sum_is_the_definition():
    """orc_direct against a numpy one-liner of eqs. (1)-(3) and field = -grad u by finite differences."""
    pos, q = inputs.uniform_cube(50, 3)
    u, f = O.direct(pos, q)
    d = pos[:, None, :] - pos[None, :, :]
    r = np.linalg.norm(d, axis=2)
    np.fill_diagonal(r, np.inf)
    want = -(q[None, :] / r).sum(axis=1) / (4 * np.pi)
    assert np.max(np.abs(u - want)) < 1e-13
    # field_i = -grad_{r_i} u(r_i) with the other charges fixed
    i, h = 7, 1e-6
    for c in range(3):
        pp, pm = pos.copy(), pos.copy()
        pp[i, c] += h
        pm[i, c] -= h
        up, _ = O.direct(pp, q, np.array([i]))
        um, _ = O.direct(pm, q, np.array([i]))
        assert abs(f[i, c] + (up[0] - um[0]) / (2 * h)) < 1e-6 * max(1.0, abs(f[i, c]))


def test_config1_error_falls_with_p():
    """BASELINE config 1: N=4096 uniform cube, q~U[-1,1], s=3, N_max=64, theta=0.77; potential+field vs O(N^2)."""
    pos, q, c = inputs.make("cfg1_cube4096_f64")
    ud, fd = O.direct(pos, q)
    prev = (1.0, 1.0)
    for p in (2, 4, 6, 8):
        P = O.Plan(pos, p, c["N_max"], c["s"], c["theta"])
        assert P.L == 2
        u, f = P.evaluate(q)
        e = (rel2(u, ud), rel2(f, fd))
        assert e[0] < 0.35 * prev[0] and e[1] < 0.45 * prev[1]
        prev = e
    assert prev[0] < 1e-5 and prev[1] < 2e-5


@pytest.mark.parametrize("N,N_max,s", [(1024, 16, 1), (2048, 8, 3)])
def test_deep_trees_error_falls_with_p(N, N_max, s):
    """deep hierarchies so that M2M and L2L carry weight (config 1 has weak pairs on its leaf level only)."""
    pos, q = inputs.uniform_cube(N, 7)
    ud, fd = O.direct(pos, q)
    prev = None
    for p in (2, 4, 6):
        P = O.Plan(pos, p, N_max, s, 0.77)
        ls = P.lists()
        nb_coarse = P.n_boxes - P.n_leaves
        assert ls["weak_off"][nb_coarse] > 0  # weak pairs above the leaf level exist
        u, f = P.evaluate(q)
        e = rel2(u, ud)
        assert prev is None or e < 0.5 * prev
        prev = e
    assert prev < 1e-3


@pytest.mark.parametrize("N,N_max,s", [(4096, 64, 3), (1024, 16, 1), (2048, 8, 3)])
def test_cross_level_lists_error_falls_with_p(N, N_max, s):
    """Level-marching lists against the O(N^2) definition: every weak pair obeys the same eq. (4), so the
    error falls with p like the same-level lists' (eq. (5)) and stays within a small factor of it, with
    fewer M2L pairs."""
    pos, q = inputs.uniform_cube(N, 7)
    ud, fd = O.direct(pos, q)
    prev = None
    for p in (2, 4, 6):
        Pc = O.Plan(pos, p, N_max, s, 0.77, cross_level=1)
        Ps = O.Plan(pos, p, N_max, s, 0.77)
        assert Pc.n_weak < Ps.n_weak and Pc.n_strong <= Ps.n_strong
        uc, fc = Pc.evaluate(q)
        us, fs = Ps.evaluate(q)
        ec, es = rel2(uc, ud), rel2(us, ud)
        assert ec < 3.0 * es and rel2(fc, fd) < 3.0 * rel2(fs, fd)
        assert prev is None or ec < 0.5 * prev
        prev = ec
    assert prev < 1e-3


def test_p0_and_all_near_field_degenerate_cases():
    pos, q = inputs.uniform_cube(300, 2)
    ud, fd = O.direct(pos, q)
    P = O.Plan(pos, 4, 512, 3)  # L = 0: root only, everything is P2P
    assert P.L == 0 and P.n_weak == 0 and P.n_strong == 1
    u, f = P.evaluate(q)
    assert rel2(u, ud) < 1e-14 and rel2(f, fd) < 1e-14
    P0 = O.Plan(pos, 0, 8, 2)  # p = 0: monopoles only, still a (crude) approximation
    u0, _ = P0.evaluate(q)
    assert rel2(u0, ud) < 0.2
    # coincident points (S3): contribute nothing to each other, result stays finite
    pos2 = np.concatenate([pos, pos[:5]], axis=0)
    q2 = np.concatenate([q, q[:5]])
    u2, f2 = O.Plan(pos2, 4, 16, 2).evaluate(q2)
    assert np.all(np.isfinite(u2)) and np.all(np.isfinite(f2))


def test_permutation_invariance():
    """tie-free input: the leaf sets do not depend on the input order (S11), results agree to rounding."""
    pos, q = inputs.uniform_cube(1500, 21)
    perm = np.random.default_rng(1).permutation(1500)
    u1, f1 = O.Plan(pos, 5, 12, 2).evaluate(q)
    u2, f2 = O.Plan(pos[perm], 5, 12, 2).evaluate(q[perm])
    assert rel2(u2, u1[perm]) < 1e-12 and rel2(f2, f1[perm]) < 1e-12


def test_masked_evaluation_equals_full_and_is_linear():
    pos, q = inputs.uniform_cube(2000, 4)
    P = O.Plan(pos, 4, 10, 2)
    u, f = P.evaluate(q)
    mask = np.zeros(P.n_leaves, np.uint8)
    mask[[0, 5, P.n_leaves - 1]] = 1
    um, fm = P.evaluate(q, leaf_mask=mask)
    sel = ~np.isnan(um)
    assert 0 < sel.sum() < 2000
    assert np.array_equal(um[sel], u[sel]) and np.array_equal(fm[sel], f[sel])
    q2 = np.random.default_rng(2).standard_normal(2000)
    ua, _ = P.evaluate(q2)
    ub, _ = P.evaluate(2.0 * q - 3.0 * q2)
    assert rel2(ub, 2.0 * u - 3.0 * ua) < 1e-12


def test_accuracy_order_of_paper_set1(golden_dir):
    """Table II set 1 (p=5, theta=0.70, N_max=128, s=2) reaches ~3 digits (8e-4 at N=2^20,
    PAPER.md:288; relative L-inf error eq. (15)).  Same order of magnitude expected on a smaller uniform cube (S1:
    the box-radius definition may differ from jaxFMM, so this is not an exact pin)."""
    vals = {l.split()[0]: float(l.split()[1]) for l in open(golden_dir + "/paper_values.txt") if l.strip() and not l.startswith("#")}
    pos, q = inputs.uniform_cube(2**13, 124)
    P = O.Plan(pos, int(vals["set1_p"]), int(vals["set1_nmax"]), int(vals["bench_s"]), vals["set1_theta"])
    u, _ = P.evaluate(q, want_field=False)
    ud, _ = O.direct(pos, q)
    err = np.max(np.abs(u - ud)) / np.max(np.abs(ud))
    assert vals["set1_err_cube"] / 30 < err < vals["set1_err_cube"] * 3


def test_p2p_pair_count_is_the_sum_over_the_strong_list():
    """orc_plan_info's n_p2p_pairs (used for the P2P roofline accounting): recomputed here from the copied lists and tree."""
    pos, _ = inputs.gaussian_clusters(6000, 8)
    for cross in (0, 1):
        P = O.Plan(pos, 4, 24, 3, 0.77, cross_level=cross)
        t, ls = P.tree(), P.lists()
        leaf0 = P.n_boxes - P.n_leaves
        cnt = t["box_count"][leaf0:]
        want = sum(int(cnt[a]) * int(cnt[ls["strong_src"][ls["strong_off"][a]:ls["strong_off"][a + 1]]].sum()) for a in range(P.n_leaves))
        assert P.n_p2p_pairs == want


def test_fp32_coincidence_rule():
    """Reading S3 for fp32 plans: the zero-distance decision is taken in binary32 (r^2 < FLT_MIN counts as coincident).  Distinct
    points 1e-23 apart: the fp64 rule sums 1/r = 1e23, the fp32 rule skips the pair; well separated points are unaffected."""
    pos = np.array([[0.0, 0.0, 0.0], [1e-23, 0.0, 0.0], [0.5, 0.25, 0.125], [0.5, 0.25, 0.125 + 2e-19]], dtype=np.float32).astype(np.float64)
    q = np.array([1.0, 2.0, -1.0, 3.0])
    u64, _ = O.direct(pos, q)
    u32, f32 = O.direct(pos, q, fp32_rule=True)
    assert abs(u64[0]) > 1e21 and abs(u32[0]) < 10 and np.all(np.isfinite(f32))
    # points 2 and 3 are 2e-19 apart in z only after rounding to binary32?  0.125 + 2e-19 rounds to 0.125: truly coincident under both rules
    assert pos[2, 2] == pos[3, 2] and abs(u64[2]) < 10
    far, qq = inputs.uniform_cube(50, 9, np.float32)
    a, b = O.direct(far, qq), O.direct(far, qq, fp32_rule=True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    P = O.Plan(pos, 3, 2, 1, 0.77)
    assert abs(P.evaluate(q, fp32_rule=True)[0][0]) < 10 and abs(P.evaluate(q)[0][0]) > 1e21
