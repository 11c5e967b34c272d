"""Pins for the oracle's hierarchy (Listing 2) and interaction lists
(PAPER.md:66-80).  Expectations come from an independent literal numpy re-enactment of Listing 2 (with its
pads), from the counts the paper states, and from brute force over all leaf pairs."""
import math

import numpy as np
import pytest

from oracle import api as O
from paper_2511_15269_b200 import inputs


def listing2_leaves(pts, max_l, s):
    """Literal re-enactment of Listing 2 in numpy.  Pad index = N; pads sort to the FRONT
    (PAPER.md:174); argpartition is replaced by a full sort in the total order (coordinate, original index)
    (reading S4); argmax returns the first maximum."""
    N = pts.shape[0]
    idcs = np.arange(N)[None, :]
    for _ in range(max_l * s):
        n = idcs.shape[1]
        needpad = n % 2
        new_rows = []
        for row in idcs:
            real = row[row < N]
            npad = len(row) - len(real)
            if len(real):
                ext = pts[real].max(axis=0) - pts[real].min(axis=0)
                ax = int(np.argmax(ext))
                order = sorted(real.tolist(), key=lambda i: (pts[i, ax], i))
            else:
                order = []
            new_rows.append([N] * npad + order + [N] * needpad)
        idcs = np.array(new_rows, dtype=np.int64).reshape((-1, (n + needpad) // 2))
    idcs = np.sort(idcs, axis=1)
    return [row[row < N].tolist() for row in idcs]


@pytest.mark.parametrize("N,N_max,s", [(37, 4, 1), (100, 3, 2), (64, 8, 3), (5, 1, 1), (200, 7, 3), (1, 4, 2), (129, 16, 2)])
def test_tree_equals_listing2(N, N_max, s):
    pos, _ = inputs.uniform_cube(N, 11)
    P = O.Plan(pos, 2, N_max, s)
    L = P.L
    # T1: smallest L with ceil(N/2^{sL}) <= N_max
    assert math.ceil(N / 2 ** (s * L)) <= N_max and (L == 0 or math.ceil(N / 2 ** (s * (L - 1))) > N_max)
    t = P.tree()
    want = listing2_leaves(pos, L, s)
    leaf0 = P.n_boxes - P.n_leaves
    got = [t["perm"][t["box_start"][leaf0 + b]: t["box_start"][leaf0 + b] + t["box_count"][leaf0 + b]].tolist() for b in range(P.n_leaves)]
    assert got == want


def test_tree_with_ties_equals_listing2():
    """lattice input: every split is a tie (config 4's situation); total order (coordinate, index), axis ties -> lowest."""
    g = np.stack(np.meshgrid(np.arange(6), np.arange(6), np.arange(3), indexing="ij"), -1).reshape(-1, 3) + 0.5
    P = O.Plan(g, 2, 4, 3)
    t = P.tree()
    want = listing2_leaves(g, P.L, 3)
    leaf0 = P.n_boxes - P.n_leaves
    got = [t["perm"][t["box_start"][leaf0 + b]: t["box_start"][leaf0 + b] + t["box_count"][leaf0 + b]].tolist() for b in range(P.n_leaves)]
    assert got == want


@pytest.mark.parametrize("N,N_max,s", [(4096, 64, 3), (1000, 16, 1), (3001, 10, 2)])
def test_tree_invariants(N, N_max, s):
    pos, _ = inputs.uniform_cube(N, 5)
    P = O.Plan(pos, 2, N_max, s)
    t = P.tree()
    assert sorted(t["perm"].tolist()) == list(range(N))  # every particle in exactly one leaf
    off = 0
    for l in range(P.L + 1):
        nb = 2 ** (s * l)
        cnt = t["box_count"][off:off + nb]
        # ceil(N/2^{ls}) or floor(N/2^{ls}) particles per box on level l
        assert set(cnt.tolist()) <= {N // nb, -(-N // nb)}
        assert cnt.sum() == N
        for b in range(nb):
            g = off + b
            ids = t["perm"][t["box_start"][g]: t["box_start"][g] + cnt[b]]
            assert np.array_equal(t["lo"][g], pos[ids].min(axis=0)) and np.array_equal(t["hi"][g], pos[ids].max(axis=0))
            assert np.array_equal(t["ctr"][g], 0.5 * (t["lo"][g] + t["hi"][g]))
            d = t["hi"][g] - t["lo"][g]
            assert t["rad"][g] == 0.5 * math.sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2])
            assert np.all(np.linalg.norm(pos[ids] - t["ctr"][g], axis=1) <= t["rad"][g] * (1 + 1e-12))
            if l > 0:  # child bbox inside parent bbox
                gp = off - 2 ** (s * (l - 1)) + b // 2**s
                assert np.all(t["lo"][g] >= t["lo"][gp]) and np.all(t["hi"][g] <= t["hi"][gp])
        off += nb
    # leaf sizes: N_max/2^s < N_box <= N_max
    leaf_cnt = t["box_count"][P.n_boxes - P.n_leaves:]
    assert leaf_cnt.max() <= N_max and leaf_cnt.min() > N_max / 2**s - 1
    # T4: ascending original index inside each leaf
    for b in range(P.n_leaves):
        g = P.n_boxes - P.n_leaves + b
        ids = t["perm"][t["box_start"][g]: t["box_start"][g] + t["box_count"][g]]
        assert np.all(np.diff(ids) > 0)


def _adm(t, a, b, theta):
    """eq. (4): R + theta r < theta d"""
    R, r = max(t["rad"][a], t["rad"][b]), min(t["rad"][a], t["rad"][b])
    return R + theta * r < theta * np.linalg.norm(t["ctr"][a] - t["ctr"][b])


@pytest.mark.parametrize("N,N_max,s,theta", [(1500, 8, 2, 0.77), (800, 6, 1, 0.5), (2048, 16, 3, 0.7)])
def test_lists_partition_identity(N, N_max, s, theta):
    """For every ordered leaf pair (t,s): exactly one of {strong; weak at exactly one ancestor level} holds,
    weak pairs satisfy eq. (4) and all their ancestors' pairs fail it; lists symmetric and sorted."""
    pos, _ = inputs.uniform_cube(N, 9)
    P = O.Plan(pos, 2, N_max, s, theta)
    t, ls = P.tree(), P.lists()
    L, nl = P.L, P.n_leaves
    off = [sum(2 ** (s * k) for k in range(l)) for l in range(L + 2)]
    weak = set()
    for g in range(P.n_boxes):
        row = ls["weak_src"][ls["weak_off"][g]: ls["weak_off"][g + 1]]
        assert np.all(np.diff(row) > 0)
        for src in row:
            weak.add((g, int(src)))
    strong = set()
    for tl in range(nl):
        row = ls["strong_src"][ls["strong_off"][tl]: ls["strong_off"][tl + 1]]
        assert np.all(np.diff(row) > 0)
        for src in row:
            strong.add((tl, int(src)))
    assert all((b, a) in weak for (a, b) in weak) and all((b, a) in strong for (a, b) in strong)
    assert all((tl, tl) in strong for tl in range(nl))
    for (a, b) in weak:
        la = max(l for l in range(L + 1) if off[l] <= a)
        assert off[la] <= b < off[la + 1]  # same level
        assert _adm(t, a, b, theta)
    rng = np.random.default_rng(0)
    pairs = [(int(a), int(b)) for a, b in rng.integers(0, nl, (4000, 2))] + [(a, a) for a in range(0, nl, 7)]
    for (a, b) in pairs:
        hits = 0
        for l in range(L + 1):
            ga, gb = off[l] + (a >> (s * (L - l))), off[l] + (b >> (s * (L - l)))
            if (ga, gb) in weak:
                hits += 1
                for k in range(l):  # all coarser ancestor pairs fail eq. (4)
                    assert not _adm(t, off[k] + (a >> (s * (L - k))), off[k] + (b >> (s * (L - k))), theta)
        if (a, b) in strong:
            assert hits == 0
            for k in range(L + 1):
                assert not _adm(t, off[k] + (a >> (s * (L - k))), off[k] + (b >> (s * (L - k))), theta)
        else:
            assert hits == 1


@pytest.mark.parametrize("N,N_max,s,theta", [(1500, 8, 2, 0.77), (800, 6, 1, 0.5), (2048, 16, 3, 0.7)])
def test_cross_level_lists_partition_identity(N, N_max, s, theta):
    """Level marching, PAPER.md:82-89 (one hierarchy for sources and targets => level pairs (0,0), (1,0), (1,1), (2,1), ...,
    (L,L)): for every ordered leaf pair (t,s) exactly one of {strong; weak at exactly one step of the march} holds; a weak
    pair satisfies eq. (4), its source sits on the target's level or one below, and the pair of every earlier step fails
    eq. (4).  (Unlike the same-level lists neither list is symmetric: the steps (l+1, l) test (coarse target, fine source)
    only, so leaf a may reach leaf b through an M2L of its parent while b sums a directly.)"""
    pos, _ = inputs.uniform_cube(N, 9)
    P = O.Plan(pos, 2, N_max, s, theta, cross_level=1)
    Ps = O.Plan(pos, 2, N_max, s, theta)
    t, ls, lss = P.tree(), P.lists(), Ps.lists()
    L, nl = P.L, P.n_leaves
    off = [sum(2 ** (s * k) for k in range(l)) for l in range(L + 2)]
    level = lambda g: max(l for l in range(L + 1) if off[l] <= g)
    anc = lambda leaf, l: off[l] + (leaf >> (s * (L - l)))
    march = [(0, 0)]
    while march[-1] != (L, L):
        lt, lsrc = march[-1]
        march.append((lt, lsrc + 1) if lsrc == lt else (lt + 1, lsrc))  # refine the sources first, then the targets
    weak = set()
    for g in range(P.n_boxes):
        row = ls["weak_src"][ls["weak_off"][g]: ls["weak_off"][g + 1]]
        assert np.all(np.diff(row) > 0)
        for src in row:
            assert level(int(src)) - level(g) in (0, 1) and _adm(t, g, int(src), theta)
            weak.add((g, int(src)))
    strong = set()
    for tl in range(nl):
        row = ls["strong_src"][ls["strong_off"][tl]: ls["strong_off"][tl + 1]]
        assert np.all(np.diff(row) > 0)
        strong.update((tl, int(src)) for src in row)
    assert all((tl, tl) in strong for tl in range(nl))
    # strong pairs fail every test of the march, in particular all same-level ones: subset of the same-level strong list
    strong_same = set()
    for tl in range(nl):
        strong_same.update((tl, int(src)) for src in lss["strong_src"][lss["strong_off"][tl]: lss["strong_off"][tl + 1]])
    assert strong <= strong_same
    assert P.n_weak < Ps.n_weak  # the point of the scheme (Table I)
    rng = np.random.default_rng(0)
    pairs = [(int(a), int(b)) for a, b in rng.integers(0, nl, (4000, 2))] + [(a, a) for a in range(0, nl, 7)]
    for (a, b) in pairs:
        hits = []
        for k, (lt, lsrc) in enumerate(march):
            if (anc(a, lt), anc(b, lsrc)) in weak:
                hits.append(k)
        if (a, b) in strong:
            assert not hits
            assert not any(_adm(t, anc(a, lt), anc(b, lsrc), theta) for (lt, lsrc) in march)
        else:
            assert len(hits) == 1
            assert not any(_adm(t, anc(a, lt), anc(b, lsrc), theta) for (lt, lsrc) in march[:hits[0]])


def test_lists_reproduce_nearest_neighbour_on_cubes(golden_dir):
    """theta = sqrt(3)/(4-sqrt(3)) ~ 0.7637 is the nearest-neighbour geometry of the uniform FMM; the
    default 0.77 reproduces it.  Hand-made geometry: 8x8x8 equal cubes (side a, radius sqrt(3)/2 a) in an octree
    numbering (s=3, L=3): interior boxes get 27 strong and 189 weak partners."""
    vals = {l.split()[0]: float(l.split()[1]) for l in open(golden_dir + "/paper_values.txt") if l.strip() and not l.startswith("#")}
    assert abs(vals["theta_nearest_neighbour"] - math.sqrt(3) / (4 - math.sqrt(3))) < 5e-5
    s, L = 3, 3
    ctr, rad = [], []
    for l in range(L + 1):
        n, a = 2**l, 1.0 / 2**l
        for b in range(8**l):
            ix = iy = iz = 0
            for k in range(l):  # octree digit k (most significant first): bits (x,y,z)
                dgt = (b >> (3 * (l - 1 - k))) & 7
                ix, iy, iz = 2 * ix + ((dgt >> 2) & 1), 2 * iy + ((dgt >> 1) & 1), 2 * iz + (dgt & 1)
            ctr.append([(ix + 0.5) * a, (iy + 0.5) * a, (iz + 0.5) * a])
            rad.append(math.sqrt(3) / 2 * a)
    nw, ns = O.lists_from_geometry(s, L, np.array(ctr), np.array(rad), vals["theta_default"])
    assert ns.max() == 27 and ns.min() == 8  # interior / corner
    leaf0 = sum(8**l for l in range(L))
    assert nw[leaf0:].max() == 189  # 6^3 - 3^3
    assert nw[0] == 0 and np.all(nw[1:9] == 0)  # nothing admissible on levels 0, 1
    # a slightly smaller theta than the nearest-neighbour value breaks the pattern (second neighbours become strong)
    nw2, ns2 = O.lists_from_geometry(s, L, np.array(ctr), np.array(rad), 0.75)
    assert ns2.max() > 27
