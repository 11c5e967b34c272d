"""Pins for the oracle's separate source / target hierarchies: the level-marching rule recomputed in numpy,
the partition identity over all (target leaf, source leaf) pairs by brute force, the reduction to the single-hierarchy
cross-level lists when both point sets coincide, and convergence to the plain definition at the targets."""
import numpy as np
import pytest

from oracle import api as O
from paper_2511_15269_b200 import inputs


def rel2(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _targets(n, seed, lo=-0.3, hi=1.4):
    return np.random.default_rng(seed).random((n, 3)) * (hi - lo) + lo


def _adm(tt, gt, ts, gs, theta):
    """eq. (4) PAPER.md:68-70 written independently in numpy"""
    R, r = max(tt["rad"][gt], ts["rad"][gs]), min(tt["rad"][gt], ts["rad"][gs])
    return R + theta * r < theta * np.linalg.norm(tt["ctr"][gt] - ts["ctr"][gs])


def _offsets(s, L):
    return [sum(2 ** (s * k) for k in range(l)) for l in range(L + 2)]


def test_direct_st_is_the_definition():
    sp, q = inputs.uniform_cube(40, 3)
    tp = _targets(25, 4)
    u, f = O.direct_st(sp, q, tp)
    d = tp[:, None, :] - sp[None, :, :]
    r = np.linalg.norm(d, axis=2)
    assert np.max(np.abs(u + (q[None, :] / r).sum(axis=1) / (4 * np.pi))) < 1e-13
    want_f = -(q[None, :, None] * d / r[:, :, None] ** 3).sum(axis=1) / (4 * np.pi)  # field = -grad u
    assert np.max(np.abs(f - want_f)) < 1e-12


@pytest.mark.parametrize("Ns,Nt,N_max,s,theta", [(1500, 700, 8, 2, 0.77), (600, 2500, 12, 1, 0.6), (2048, 2048, 16, 3, 0.7)])
def test_march_follows_the_mean_radius_rule_and_partitions_all_leaf_pairs(Ns, Nt, N_max, s, theta):
    sp, _ = inputs.uniform_cube(Ns, 21)
    tp = _targets(Nt, 22)
    P = O.PlanST(sp, tp, 2, N_max, s, theta)
    ts, tt, ls = P.tree("src"), P.tree("tgt"), P.lists()
    Ls, Lt = P.info["src"]["L"], P.info["tgt"]["L"]
    offs, offt = _offsets(s, Ls), _offsets(s, Lt)

    def mean_rad(t, off, l):
        sel = t["box_count"][off[l]:off[l + 1]] > 0
        return t["rad"][off[l]:off[l + 1]][sel].mean()

    # PAPER.md:85-88 re-enacted: refine the level with the larger mean radius; ties -> source; exhausted side -> the other
    steps = [(0, 0)]
    while steps[-1] != (Lt, Ls):
        lt, lsrc = steps[-1]
        if lsrc == Ls:
            steps.append((lt + 1, lsrc))
        elif lt == Lt:
            steps.append((lt, lsrc + 1))
        else:
            rt, rs = mean_rad(tt, offt, lt), mean_rad(ts, offs, lsrc)
            assert abs(rt - rs) > 1e-9 * max(rt, rs)  # no near-tie, so numpy's summation order cannot flip the decision
            steps.append((lt + 1, lsrc) if rt > rs else (lt, lsrc + 1))
    assert ls["steps"].tolist() == [list(x) for x in steps]

    level_t = lambda g: max(l for l in range(Lt + 1) if offt[l] <= g)
    level_s = lambda g: max(l for l in range(Ls + 1) if offs[l] <= g)
    weak = set()
    for g in range(P.info["tgt"]["n_boxes"]):
        row = ls["weak_src"][ls["weak_off"][g]: ls["weak_off"][g + 1]]
        assert np.all(np.diff(row) > 0)
        for src in row:
            assert (level_t(g), level_s(int(src))) in steps and _adm(tt, g, ts, int(src), theta)
            weak.add((g, int(src)))
    strong = set()
    nlt, nls = P.info["tgt"]["n_leaves"], P.info["src"]["n_leaves"]
    for tl in range(nlt):
        row = ls["strong_src"][ls["strong_off"][tl]: ls["strong_off"][tl + 1]]
        assert np.all(np.diff(row) > 0)
        strong.update((tl, int(src)) for src in row)
    anc_t = lambda leaf, l: offt[l] + (leaf >> (s * (Lt - l)))
    anc_s = lambda leaf, l: offs[l] + (leaf >> (s * (Ls - l)))
    rng = np.random.default_rng(0)
    pairs = list(zip(rng.integers(0, nlt, 3000).tolist(), rng.integers(0, nls, 3000).tolist()))
    for (a, b) in pairs:
        if tt["box_count"][offt[Lt] + a] == 0 or ts["box_count"][offs[Ls] + b] == 0:
            continue
        hits = [k for k, (lt, lsrc) in enumerate(steps) if (anc_t(a, lt), anc_s(b, lsrc)) in weak]
        if (a, b) in strong:
            assert not hits and not any(_adm(tt, anc_t(a, lt), ts, anc_s(b, lsrc), theta) for (lt, lsrc) in steps)
        else:  # covered exactly once, at the first step of the march whose ancestor pair is admissible
            assert len(hits) == 1
            assert not any(_adm(tt, anc_t(a, lt), ts, anc_s(b, lsrc), theta) for (lt, lsrc) in steps[:hits[0]])


@pytest.mark.parametrize("N,N_max,s", [(3000, 32, 2), (37, 1, 2), (150, 1, 3), (9, 1, 1)])
def test_identical_sets_reduce_to_the_single_hierarchy_cross_level_lists(N, N_max, s):
    """Sources == targets: both hierarchies coincide, mean radii tie on equal levels (-> source first), so the march is the fixed
    sequence (l_trg, l_src) = (0,0), (0,1), (1,1), (1,2), ... of the single-hierarchy cross-level plan and lists and results must
    be identical -- also on ragged trees (N < 2^(sL): empty boxes, levels whose mean radius is taken over the non-empty boxes only)."""
    pos, q = inputs.uniform_cube(N, 5)
    P1 = O.Plan(pos, 5, N_max, s, 0.77, cross_level=1)
    P2 = O.PlanST(pos, pos, 5, N_max, s, 0.77)
    assert N_max > 1 or N < 2 ** (s * P1.L)  # the small cases are ragged
    l1, l2 = P1.lists(), P2.lists()
    for k in ("weak_off", "weak_src", "strong_off", "strong_src"):
        assert np.array_equal(l1[k], l2[k])
    want = [(0, 0)]
    while want[-1] != (P1.L, P1.L):
        lt, ls = want[-1]
        want.append((lt, ls + 1) if lt == ls else (lt + 1, ls))
    assert [tuple(x) for x in l2["steps"]] == want
    u1, f1 = P1.evaluate(q)
    u2, f2 = P2.evaluate(q)
    # the single-set evaluate skips the pair i == j by index, the two-set evaluate by distance: same terms, same order
    assert np.array_equal(u1, u2) and np.array_equal(f1, f2)


def test_masked_evaluation_st_equals_full():
    """leaf mask of evaluate_st (used by the full-size GPU parity tests): the masked target leaves get bit-for-bit the values of a
    full run, every other target stays untouched."""
    sp, q = inputs.uniform_cube(3000, 61)
    tp = _targets(2200, 62)
    P = O.PlanST(sp, tp, 6, 16, 2, 0.77)
    u, f = P.evaluate(q)
    nl = P.info["tgt"]["n_leaves"]
    mask = np.zeros(nl, np.uint8)
    mask[np.random.default_rng(3).choice(nl, 9, replace=False)] = 1
    um, fm = P.evaluate(q, leaf_mask=mask)
    t = P.tree("tgt")
    off = _offsets(2, P.info["tgt"]["L"])[P.info["tgt"]["L"]]
    sel = np.concatenate([t["perm"][t["box_start"][off + l]: t["box_start"][off + l] + t["box_count"][off + l]] for l in np.flatnonzero(mask)])
    assert sel.size > 0 and np.array_equal(um[sel], u[sel]) and np.array_equal(fm[sel], f[sel])
    rest = np.setdiff1d(np.arange(tp.shape[0]), sel)
    assert np.all(np.isnan(um[rest])) and np.all(np.isnan(fm[rest]))


@pytest.mark.parametrize("Ns,Nt,N_max,s", [(3000, 2000, 32, 2), (1024, 4096, 16, 3)])
def test_separate_targets_error_falls_with_p(Ns, Nt, N_max, s):
    sp, q = inputs.uniform_cube(Ns, 31)
    tp = _targets(Nt, 32)
    ud, fd = O.direct_st(sp, q, tp)
    errs = []
    for p in (2, 4, 6, 8):
        u, f = O.PlanST(sp, tp, p, N_max, s, 0.77).evaluate(q)
        errs.append((rel2(u, ud), rel2(f, fd)))
    for a, b in zip(errs, errs[1:]):
        assert b[0] < 0.5 * a[0] and b[1] < 0.6 * a[1], errs
    assert errs[-1][0] < 5e-4 and errs[-1][1] < 5e-4, errs


def test_targets_far_from_all_sources_use_the_root_multipole():
    """Degenerate march: every target box is admissible against the source root at the first refinement -> one weak pair per
    target box of that level, no strong pair; result equals the definition to the truncation error of a far expansion."""
    sp, q = inputs.uniform_cube(500, 41)
    tp = _targets(300, 42, 20.0, 21.0)
    P = O.PlanST(sp, tp, 8, 16, 2, 0.77)
    assert P.n_strong == 0 and P.n_weak >= 1
    u, f = P.evaluate(q)
    ud, fd = O.direct_st(sp, q, tp)
    assert rel2(u, ud) < 1e-9 and rel2(f, fd) < 1e-8
