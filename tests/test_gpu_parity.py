"""GPU parity tests proper: the CUDA path (through the C-ABI binding) against the CPU oracle on the same seeded inputs.

Acceptance (BASELINE.json north_star): hierarchy and interaction lists bit-exact; rel-L2(GPU - oracle) <= 1e-5 (fp32) and
<= 1e-11 (fp64) on potential and on field at equal p; error against the O(N^2) definition within 1.5x the oracle's own.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs

pytestmark = pytest.mark.gpu

TOL = {np.float32: 1e-5, np.float64: 1e-11}  # north_star tolerances, rel-L2 GPU vs oracle
# Element-wise bound, max_i |gpu_i - oracle_i| / max_i |oracle_i|: a single output is a sum of ~1e3 near-field
# terms and ~2e2 x L translated expansions of both signs; with unit roundoff u (6e-8 / 1.1e-16) and random-sign accumulation its
# error relative to the largest output is a few 10 u sqrt(terms) ~ 100 u in the bulk, up to ~10x that at the worst of 1e6 outputs.
TOL_MAX = {np.float32: 1e-4, np.float64: 1e-10}


def rel2(a, b):
    return np.linalg.norm(np.asarray(a, np.float64) - b) / np.linalg.norm(b)


def gpu_plan(pos, p, N_max, s, theta=0.77, cross_level=0):
    tp = torch.from_numpy(np.ascontiguousarray(pos)).cuda()
    return fmm.Plan(tp, p, N_max, s, theta, cross_level=cross_level)


def gpu_eval(P, q):
    tq = torch.from_numpy(np.ascontiguousarray(q)).cuda()
    u, f = P.evaluate(tq)
    torch.cuda.synchronize()
    return u.cpu().numpy(), f.cpu().numpy()


def assert_same_hierarchy(P, Po, dtype):
    """bit-exact: permutation, box ranges, tight boxes, fp64 centres/radii, both lists in canonical CSR form."""
    tg, to = P.tree(), Po.tree()
    info = P.info
    assert (info["L"], info["n_boxes"], info["n_leaves"]) == (Po.L, Po.n_boxes, Po.n_leaves)
    assert np.array_equal(tg["perm"].astype(np.int64), to["perm"])
    assert np.array_equal(tg["box_count"].astype(np.int64), to["box_count"])
    ne = to["box_count"] > 0
    assert np.array_equal(tg["box_start"].astype(np.int64)[ne], to["box_start"][ne])
    assert np.array_equal(tg["lo"].astype(np.float64)[ne], to["lo"][ne])
    assert np.array_equal(tg["hi"].astype(np.float64)[ne], to["hi"][ne])
    assert np.array_equal(tg["ctr"][ne], to["ctr"][ne])  # fp64, no FMA contraction on either side (rule T6)
    assert np.array_equal(tg["rad"][ne], to["rad"][ne])
    lg, lo_ = P.lists(), Po.lists()
    assert (info["n_weak"], info["n_strong"], info["n_p2p_pairs"]) == (Po.n_weak, Po.n_strong, Po.n_p2p_pairs)
    assert np.array_equal(lg["weak_off"], lo_["weak_off"])
    assert np.array_equal(lg["weak_src"].astype(np.int64), lo_["weak_src"])
    assert np.array_equal(lg["strong_off"], lo_["strong_off"])
    assert np.array_equal(lg["strong_src"].astype(np.int64), lo_["strong_src"])


def relmax(a, b):
    return np.max(np.abs(np.asarray(a, np.float64) - b)) / np.max(np.abs(b))


def run_case(pos, q, p, N_max, s, theta=0.77, direct=True):
    dt = pos.dtype.type
    f32 = dt == np.float32  # the zero-distance decision (reading S3) is taken in the plan's precision on both sides
    P = gpu_plan(pos, p, N_max, s, theta)
    Po = O.Plan(pos, p, N_max, s, theta)
    assert_same_hierarchy(P, Po, dt)
    u, f = gpu_eval(P, q)
    uo, fo = Po.evaluate(q, fp32_rule=f32)
    assert np.all(np.isfinite(u)) and np.all(np.isfinite(f))
    eu, ef = rel2(u, uo), rel2(f, fo)
    assert eu <= TOL[dt] and ef <= TOL[dt], (eu, ef)
    assert relmax(u, uo) <= TOL_MAX[dt] and relmax(f, fo) <= TOL_MAX[dt], (relmax(u, uo), relmax(f, fo))
    if direct:
        ud, fd = O.direct(pos, q, fp32_rule=f32)
        assert rel2(u, ud) <= 1.5 * rel2(uo, ud) + 1e-14
        assert rel2(f, fd) <= 1.5 * rel2(fo, fd) + 1e-14
    P.close()
    return eu, ef


# ------------------------------------------------------------------------------------------- BASELINE config 1
def test_config1_fp64():
    pos, q, c = inputs.make("cfg1_cube4096_f64")
    run_case(pos, q, c["p"], c["N_max"], c["s"], c["theta"])


def test_config1_shape_fp32():
    pos, q = inputs.uniform_cube(4096, 1, np.float32)
    run_case(pos, q, 6, 64, 3)


# ------------------------------------------------------------------------------------------- deep trees (M2M / L2L carry weight)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s,p", [(1024, 16, 1, 6), (4096, 8, 3, 4), (3000, 20, 2, 8), (5000, 40, 1, 5)])
def test_deep_trees(dtype, N, N_max, s, p):
    pos, q = inputs.uniform_cube(N, 7, dtype)
    run_case(pos, q, p, N_max, s)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("p", [0, 1, 2, 3, 7, 9, 10, 11, 12, 13, 14, 15, 16])
def test_orders(dtype, p):
    """every order the header accepts (0 .. FMM_P_MAX = 16) on a deep tree (L = 4): p <= 8 register kernels, 9..12 shared-memory
    kernels, 13..16 the generic warp-per-box kernels."""
    pos, q = inputs.uniform_cube(2500, 11, dtype)
    run_case(pos, q, p, 32, 2)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("p", [13, 16])
def test_highest_orders_clusters_and_generic_family(dtype, p):
    """p = 13..16 are served by the generic kernels in both kernel families; non-uniform input, s = 3, cross-level lists too."""
    pos, q = inputs.gaussian_clusters(4000, 15, dtype)
    run_case(pos, q, p, 24, 3)
    P = gpu_plan(pos, p, 24, 3, 0.77, cross_level=1)
    Po = O.Plan(pos, p, 24, 3, 0.77, cross_level=1)
    fmm.fmm_plan_set_m2l_variant(P.handle, 1)
    u, f = gpu_eval(P, q)
    uo, fo = Po.evaluate(q, fp32_rule=dtype == np.float32)
    assert rel2(u, uo) <= TOL[dtype] and rel2(f, fo) <= TOL[dtype]
    P.close()


@pytest.mark.parametrize("theta", [0.3, 0.5, 0.9])
def test_theta(theta):
    pos, q = inputs.uniform_cube(3000, 12, np.float64)
    run_case(pos, q, 6, 24, 3, theta)


# ------------------------------------------------------------------------------------------- other point distributions
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_sphere_surface(dtype):
    pos, q = inputs.sphere_surface(6000, 21, dtype)
    run_case(pos, q, 8, 32, 3)


@pytest.mark.parametrize("dtype,s", [(np.float64, 3), (np.float32, 3), (np.float32, 1)])
def test_clusters(dtype, s):
    pos, q = inputs.gaussian_clusters(20000, 3, dtype)
    run_case(pos, q, 8, 48, s)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_thin_film_lattice_all_ties(dtype):
    """config-4 shape at reduced size: every coordinate is tied many times (reading S4 decides the tree)."""
    pos, q = inputs.thin_film(64, 48, 4, 4, dtype)
    run_case(pos, q, 6, 16, 3)


# ------------------------------------------------------------------------------------------- degenerate inputs
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s", [(1, 4, 3), (2, 1, 1), (5, 8, 3), (7, 1, 3), (9, 1, 2), (100, 128, 3), (129, 128, 3), (1000, 1, 1)])
def test_tiny_and_ragged(dtype, N, N_max, s):
    """L = 0 (root only, all P2P), N < 2^(sL) (empty boxes, rule T5), one particle per leaf."""
    pos, q = inputs.uniform_cube(N, 100 + N, dtype)
    P = gpu_plan(pos, 4, N_max, s)
    Po = O.Plan(pos, 4, N_max, s)
    assert_same_hierarchy(P, Po, dtype)
    u, f = gpu_eval(P, q)
    uo, fo = Po.evaluate(q, fp32_rule=dtype == np.float32)
    if N == 1:
        assert u[0] == 0 and np.all(f == 0)
    else:
        assert rel2(u, uo) <= TOL[dtype] and rel2(f, fo) <= TOL[dtype]
    P.close()


def test_coincident_points_contribute_nothing():
    """reading S3: zero-distance pairs are skipped (potential and field stay finite)."""
    pos, q = inputs.uniform_cube(600, 5, np.float64)
    pos[100:140] = pos[0:40]
    run_case(pos, q, 5, 16, 2)


@pytest.mark.parametrize("variant", [0, 1])
def test_fp32_distances_that_underflow(variant):
    """Reading S3, fp32 clause: distinct points whose squared distance is below FLT_MIN in binary32 (here 5e-20 .. 7e-20 apart)
    count as coincident on both sides (the oracle takes the decision in binary32 too); both kernel families; everything finite."""
    pos, q = inputs.uniform_cube(800, 19, np.float32)
    rng = np.random.default_rng(20)
    # 8 pairs near the origin (binary32 resolves 1e-19 only there): the bases on a 2 x 2 x 2 lattice of spacing 3e-13 -- far enough apart
    # for q / r^3 < FLT_MAX, which the fp32 field arithmetic needs (reading S3) -- the partner of each 5e-20 .. 7e-20 away in x:
    # a distinct binary32 point whose r^2 (<= 5e-39) is below FLT_MIN.
    base = np.array([[i, j, k] for i in (0, 1) for j in (0, 1) for k in (0, 1)], dtype=np.float64) * 3e-13
    part = base.astype(np.float32).copy()
    part[:, 0] = np.where(part[:, 0] == 0, np.float32(5e-20), np.nextafter(np.nextafter(part[:, 0], np.float32(1)), np.float32(1)))
    pos[:8] = base.astype(np.float32)
    pos[8:16] = part
    gap = pos[8:16, 0].astype(np.float64) - pos[:8, 0]
    assert np.all(gap > 0) and np.all(gap * gap < 1.1754944e-38)  # distinct points, r^2 not a normal binary32 number
    q = q.copy()
    q[:16] = rng.uniform(0.5, 1.0, 16).astype(np.float32)
    P = gpu_plan(pos, 5, 16, 2)
    Po = O.Plan(pos, 5, 16, 2)
    assert_same_hierarchy(P, Po, np.float32)
    fmm.fmm_plan_set_m2l_variant(P.handle, variant)
    u, f = gpu_eval(P, q)
    uo, fo = Po.evaluate(q, fp32_rule=True)
    assert np.all(np.isfinite(u)) and np.all(np.isfinite(f))
    assert rel2(u, uo) <= 1e-5 and rel2(f, fo) <= 1e-5, (rel2(u, uo), rel2(f, fo))
    u64, _ = Po.evaluate(q)  # the fp64 rule sums 1/r ~ 1e20 for those pairs: the two readings really differ on this input
    assert np.max(np.abs(u64)) > 1e3 * np.max(np.abs(uo))
    P.close()


def test_collinear_and_planar_points():
    """boxes with zero extent along one or two axes; translations along +-z and in the xy-plane (reading S7)."""
    rng = np.random.default_rng(9)
    z = np.zeros((800, 3))
    z[:, 2] = rng.random(800)
    run_case(z, rng.uniform(-1, 1, 800), 6, 16, 1)
    xy = rng.random((1500, 3))
    xy[:, 2] = 0.25
    run_case(xy, rng.uniform(-1, 1, 1500), 6, 16, 2)


def test_small_and_large_length_scales_fp32():
    """hard part 1 of DESIGN.md: unscaled fp32 coefficients would overflow/underflow; the scaled representation must not."""
    for scale in (1e-4, 1.0, 1e4):
        pos, q = inputs.uniform_cube(4000, 13, np.float64)
        pos = (pos * scale).astype(np.float32)
        run_case(pos, q.astype(np.float32), 8, 16, 3)


def test_plan_reuse_and_linearity():
    """one hierarchy, many charge vectors; the evaluate is linear in q."""
    pos, q1 = inputs.uniform_cube(3000, 30, np.float64)
    _, q2 = inputs.uniform_cube(3000, 31, np.float64)
    P = gpu_plan(pos, 6, 32, 3)
    u1, f1 = gpu_eval(P, q1)
    u2, f2 = gpu_eval(P, q2)
    u3, f3 = gpu_eval(P, 2.0 * q1 - 3.0 * q2)
    assert rel2(u3, 2.0 * u1 - 3.0 * u2) < 1e-12 and rel2(f3, 2.0 * f1 - 3.0 * f2) < 1e-12
    u1b, f1b = gpu_eval(P, q1)
    # repeatable to rounding: the register translation kernels accumulate M2L/L2L results with atomics, whose order varies
    assert rel2(u1b, u1) < 1e-13 and rel2(f1b, f1) < 1e-13
    P.close()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("gen,N,N_max,s,p,cross", [("cube", 20000, 32, 3, 8, 0), ("cube", 6000, 16, 2, 6, 1), ("clusters", 30000, 48, 1, 5, 0),
                                                    ("cube", 3000, 20, 2, 10, 0), ("cube", 1500, 512, 3, 4, 0)])
def test_deterministic_mode_is_bit_for_bit_reproducible(dtype, gen, N, N_max, s, p, cross):
    """fmm_plan_set_deterministic: two evaluates of the same charges return identical bits (no float atomics with several contributors,
    serial schedule), the result still meets the parity tolerance, and switching the mode off again restores the default kernels."""
    pos, q = (inputs.uniform_cube if gen == "cube" else inputs.gaussian_clusters)(N, 41, dtype)
    P = gpu_plan(pos, p, N_max, s, 0.77, cross_level=cross)
    Po = O.Plan(pos, p, N_max, s, 0.77, cross_level=cross)
    uo, fo = Po.evaluate(q, fp32_rule=dtype == np.float32)
    fmm.fmm_plan_set_deterministic(P.handle, 1)
    runs = [gpu_eval(P, q) for _ in range(4)]
    for u, f in runs[1:]:
        assert np.array_equal(u, runs[0][0]) and np.array_equal(f, runs[0][1])
    assert rel2(runs[0][0], uo) <= TOL[dtype] and rel2(runs[0][1], fo) <= TOL[dtype]
    u2, f2 = gpu_eval(P, -q)  # another charge vector in between must not leave anything behind
    u3, f3 = gpu_eval(P, q)
    assert np.array_equal(u3, runs[0][0]) and np.array_equal(f3, runs[0][1]) and np.array_equal(u2, -runs[0][0])
    fmm.fmm_plan_set_deterministic(P.handle, 0)
    u, f = gpu_eval(P, q)
    assert rel2(u, uo) <= TOL[dtype] and rel2(f, fo) <= TOL[dtype]
    P.close()


@pytest.mark.parametrize("N,N_max,s,p", [(4096, 64, 3, 8), (3001, 8, 3, 8), (5000, 40, 1, 5), (2000, 16, 2, 1)])
def test_kernel_families_agree_with_the_oracle_fp32(N, N_max, s, p):
    """fmm_plan_set_m2l_variant: the one-translation-per-thread kernels (0) and the generic warp-per-box kernels (1) are two
    independent implementations of App. B; each must meet the fp32 tolerance against the oracle on its own."""
    pos, q = inputs.uniform_cube(N, 11, np.float32)
    Po = O.Plan(pos, p, N_max, s, 0.77)
    uo, fo = Po.evaluate(q)
    P = gpu_plan(pos, p, N_max, s)
    for variant in (0, 1):
        fmm.fmm_plan_set_m2l_variant(P.handle, variant)
        u, f = gpu_eval(P, q)
        assert rel2(u, uo) <= 1e-5 and rel2(f, fo) <= 1e-5, (variant, rel2(u, uo), rel2(f, fo))
    P.close()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s,p,theta", [(4096, 64, 3, 6, 0.77), (1024, 16, 1, 6, 0.77), (4096, 8, 3, 4, 0.5), (3000, 20, 2, 8, 0.77),
                                                (5, 8, 3, 4, 0.77), (129, 128, 3, 3, 0.77), (1000, 1, 1, 2, 0.77)])
def test_cross_level_lists(dtype, N, N_max, s, p, theta):
    """cross_level = 1 (level marching): hierarchy and both lists bit-exact against the oracle's, potential and
    field within the north_star tolerance of the oracle evaluated on the same lists, and fewer weak pairs than same-level."""
    pos, q = inputs.uniform_cube(N, 21, dtype)
    P = gpu_plan(pos, p, N_max, s, theta, cross_level=1)
    Po = O.Plan(pos, p, N_max, s, theta, cross_level=1)
    assert_same_hierarchy(P, Po, dtype)
    u, f = gpu_eval(P, q)
    uo, fo = Po.evaluate(q)
    assert rel2(u, uo) <= TOL[dtype] and rel2(f, fo) <= TOL[dtype]
    if Po.L >= 2:
        assert P.info["n_weak"] < O.Plan(pos, p, N_max, s, theta).n_weak
    if dtype == np.float32:
        for variant in (1,):
            fmm.fmm_plan_set_m2l_variant(P.handle, variant)
            u, f = gpu_eval(P, q)
            assert rel2(u, uo) <= TOL[dtype] and rel2(f, fo) <= TOL[dtype], variant
    P.close()


def test_cross_level_clusters_and_lattice_fp32():
    """non-uniform and all-ties inputs through the marching builder (stable sort by target must keep sources ascending)"""
    for name, n in (("clusters", 30000), ("film", 0)):
        if name == "clusters":
            pos, q = inputs.gaussian_clusters(n, 5, np.float32)
            args = (8, 32, 3)
        else:
            pos, q = inputs.thin_film(32, 32, 4, 6, np.float32)
            args = (6, 16, 3)
        P = gpu_plan(pos, *args, cross_level=1)
        Po = O.Plan(pos, *args, cross_level=1)
        assert_same_hierarchy(P, Po, np.float32)
        u, f = gpu_eval(P, q)
        uo, fo = Po.evaluate(q)
        assert rel2(u, uo) <= 1e-5 and rel2(f, fo) <= 1e-5
        P.close()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_concurrent_and_serial_schedules_agree(dtype):
    """fmm_plan_set_schedule: the forked-stream schedule (default) and the single-stream schedule run the same kernels;
    both must meet the tolerance, repeatedly on one plan (stream joins must order consecutive evaluates), also on a side stream."""
    pos, q = inputs.uniform_cube(20000, 12, dtype)
    p = 8 if dtype == np.float32 else 6
    Po = O.Plan(pos, p, 32, 3, 0.77)
    uo, fo = Po.evaluate(q)
    P = gpu_plan(pos, p, 32, 3)
    for serial in (0, 1, 0):
        fmm.fmm_plan_set_schedule(P.handle, serial)
        for rep in range(3):
            u, f = gpu_eval(P, q if rep != 1 else -q)
            sgn = 1.0 if rep != 1 else -1.0
            assert rel2(sgn * u, uo) <= TOL[dtype] and rel2(sgn * f, fo) <= TOL[dtype], (serial, rep)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        tq = torch.from_numpy(q).cuda()
        u, f = P.evaluate(tq)
    side.synchronize()
    assert rel2(u.cpu().numpy(), uo) <= TOL[dtype]
    P.close()


def test_potential_only_and_field_only_and_host_path():
    pos, q = inputs.uniform_cube(2000, 33, np.float32)
    P = gpu_plan(pos, 5, 32, 3)
    u, f = gpu_eval(P, q)
    tq = torch.from_numpy(q).cuda()
    u2, none = P.evaluate(tq, want_field=False)
    none2, f2 = P.evaluate(tq, want_potential=False)
    torch.cuda.synchronize()
    assert none is None and none2 is None
    # the fp32 register translation kernels add partial sums with atomicAdd, so repeated runs agree to rounding only
    assert rel2(u2.cpu().numpy(), u.astype(np.float64)) < 2e-6 and rel2(f2.cpu().numpy(), f.astype(np.float64)) < 2e-6
    hu, hf = np.empty_like(u), np.empty_like(f)
    fmm.fmm_evaluate_host(P.handle, q, hu, hf)
    assert rel2(hu, u.astype(np.float64)) < 2e-6 and rel2(hf, f.astype(np.float64)) < 2e-6
    P.close()


def test_non_finite_positions_are_rejected():
    pos, _ = inputs.uniform_cube(100, 1, np.float32)
    pos[17, 1] = np.nan
    with pytest.raises(fmm.FmmError) as e:
        gpu_plan(pos, 4, 16, 2)
    assert e.value.status == fmm.FMM_ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------- full-size configs (sampled oracle)
def sampled_case(name, n_sample_leaves=12, seed=0, cross_level=0, workload=None, n_direct_targets=0):
    """BASELINE full-size configs in the configuration bench.py times: hierarchy/lists bit-exact on everything;
    potential/field compared on the particles of a random sample of leaves (the oracle computes exactly those,
    with the same arithmetic as a full run): rel-L2 AND element by element; and against the O(N^2) definition on the same
    particles.  n_direct_targets > 0 adds SURVEY 8(c)'s acceptance clause as written: that many random targets against all N
    sources, error of the GPU result <= 1.5 x the oracle's."""
    pos, q, c = inputs.make(name) if workload is None else workload
    dt = pos.dtype.type
    f32 = dt == np.float32
    P = gpu_plan(pos, c["p"], c["N_max"], c["s"], c["theta"], cross_level=cross_level)
    Po = O.Plan(pos, c["p"], c["N_max"], c["s"], c["theta"], cross_level=cross_level)
    assert_same_hierarchy(P, Po, dt)
    u, f = gpu_eval(P, q)
    assert np.all(np.isfinite(u)) and np.all(np.isfinite(f))
    rng = np.random.default_rng(seed)
    mask = np.zeros(Po.n_leaves, np.uint8)
    mask[rng.choice(Po.n_leaves, n_sample_leaves, replace=False)] = 1
    tgt = None
    if n_direct_targets:
        tgt = np.sort(rng.choice(pos.shape[0], n_direct_targets, replace=False))
        t = Po.tree()
        leaf0 = Po.n_boxes - Po.n_leaves
        inv = np.empty(pos.shape[0], np.int64)
        inv[t["perm"]] = np.arange(pos.shape[0])
        mask[np.searchsorted(t["box_start"][leaf0:], inv[tgt], side="right") - 1] = 1  # the leaves holding the random targets
    uo, fo = Po.evaluate(q, leaf_mask=mask, fp32_rule=f32)
    sel = np.flatnonzero(np.isfinite(uo))
    assert sel.size > 0
    eu, ef = rel2(u[sel], uo[sel]), rel2(f[sel], fo[sel])
    assert eu <= TOL[dt] and ef <= TOL[dt], (eu, ef)
    mu, mf = relmax(u[sel], uo[sel]), relmax(f[sel], fo[sel])
    assert mu <= TOL_MAX[dt] and mf <= TOL_MAX[dt], (mu, mf)
    if tgt is None:
        dsel = sel if sel.size <= 4096 else np.sort(rng.choice(sel, 4096, replace=False))
    else:
        assert np.all(np.isfinite(uo[tgt]))
        dsel = tgt
    ud, fd = O.direct(pos, q, dsel, fp32_rule=f32)
    assert rel2(u[dsel], ud) <= 1.5 * rel2(uo[dsel], ud)
    assert rel2(f[dsel], fd) <= 1.5 * rel2(fo[dsel], fd)
    P.close()
    return dict(n_weak=Po.n_weak, n_compared=int(sel.size), err_u=rel2(u[dsel], ud), err_f=rel2(f[dsel], fd), err_u_oracle=rel2(uo[dsel], ud),
                err_f_oracle=rel2(fo[dsel], fd), gpu_vs_oracle=(eu, ef, mu, mf))


def test_config2_full_size_sampled():
    """headline configuration: 256 random leaves (~7 800 particles) compared element by element, plus SURVEY 8(c)'s acceptance
    clause -- 2048 random targets against all 1e6 sources through the plain definition."""
    r = sampled_case("cfg2_cube1M_f32", n_sample_leaves=256, n_direct_targets=2048)
    print("cfg2", r)
    assert r["n_compared"] > 7000


@pytest.mark.parametrize("name,nl,slack", [("cfg2_cube1M_f32", 12, 3.0), ("cfg3_clusters1M_f32_s3", 8, 3.0), ("cfg4_film_f32", 24, 10.0)])
def test_full_size_sampled_cross_level(name, nl, slack):
    """level-marching lists at full size: same acceptance as the same-level lists (GPU == oracle on the same lists, error vs
    the O(N^2) definition within 1.5x the oracle's).  Against the same-level lists at equal theta the scheme itself trades
    accuracy for pairs: measured on B200, -42 % pairs / 1.6x the error (uniform cube), -51 % / 1.5x (clusters),
    -62 % / 7x (lattice with tight boxes, p = 6); the bound here only guards the order of magnitude."""
    rc = sampled_case(name, n_sample_leaves=nl, cross_level=1)
    rs = sampled_case(name, n_sample_leaves=nl, cross_level=0)
    print(name, "cross", rc, "same", rs)
    assert rc["n_weak"] < 0.7 * rs["n_weak"]
    assert rc["err_u"] < slack * rs["err_u"] and rc["err_f"] < slack * rs["err_f"]


@pytest.mark.parametrize("name,nl", [("cfg3_clusters1M_f32_s3", 64), ("cfg3_clusters1M_f32_s1", 24)])
def test_config3_full_size_sampled(name, nl):
    sampled_case(name, n_sample_leaves=nl)


def test_config4_full_size_sampled():
    sampled_case("cfg4_film_f32", n_sample_leaves=128)


def test_config5_ten_million_sampled():
    """Largest N of BASELINE config 5 (N = 1e7, uniform cube, fp32, p = 8, N_max = 128, s = 3): 2.4e5 leaves, 5.6e7 weak pairs --
    hierarchy and both lists bit-exact, potential/field on the particles of 4 sampled leaves."""
    pos, q = inputs.uniform_cube(10**7, 57, np.float32)
    sampled_case("cfg5_cube1e7_f32", n_sample_leaves=32, workload=(pos, q, dict(p=8, N_max=128, s=3, theta=0.77)))


def test_config5_sphere_one_million_sampled():
    """Config 5, points on the unit-sphere surface, N = 1e6, fp32, p = 8."""
    pos, q = inputs.sphere_surface(10**6, 56, np.float32)
    sampled_case("cfg5_sphere1e6_f32", n_sample_leaves=64, workload=(pos, q, dict(p=8, N_max=128, s=3, theta=0.77)))


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s,p", [(20000, 512, 3, 6), (5000, 512, 1, 4), (3000, 3000, 2, 5)])
def test_large_leaves(dtype, N, N_max, s, p):
    """Config 5's N_max = 512: leaves of 300+ particles are cut into chunks of 32 x TPT targets per warp (P2P), several
    P2M / L2P passes per leaf; N_max >= N gives a single leaf (L = 0, everything is P2P)."""
    pos, q = inputs.uniform_cube(N, 58, dtype)
    run_case(pos, q, p, N_max, s, direct=N_max < N)  # a single leaf: the oracle IS the direct sum, nothing to compare the error with
