"""fmm_evaluate_adjoint: gradient of a loss on potential / field with respect to the charges (PAPER.md:281-310,
"Active Shielding").

The evaluate is linear in the charges, potential = A q and field = F q with the FMM operators of the plan, so the vector-Jacobian
product the paper obtains by JAX autodiff is q_bar = A^T u_bar + F^T f_bar.  The library computes it as the transpose of the forward
operator on the SAME plan (transposed lists, M2M <-> L2L, P2M <-> L2P, dipole sources for the field part); the oracle's
evaluate_adjoint is the same transposition written plainly (tests/test_oracle_adjoint.py pins it).  Here: device vs oracle at the
north_star tolerance, the dot-product identity against the device's own forward evaluate to ROUNDING level, and the paper's
shielding demo driven through the C-ABI only."""
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
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def fib_sphere(n, r):
    """n points spread evenly on a sphere of radius r (golden-angle spiral)"""
    k = np.arange(n) + 0.5
    z = 1.0 - 2.0 * k / n
    ph = np.pi * (1.0 + 5.0 ** 0.5) * k
    s = np.sqrt(1.0 - z * z)
    return np.ascontiguousarray(r * np.stack([s * np.cos(ph), s * np.sin(ph), z], axis=1))


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("N,N_max,s,p,cross", [(1500, 32, 2, 6, 0), (1500, 32, 2, 6, 1), (4096, 8, 3, 4, 1), (500, 20, 1, 8, 0), (250, 16, 2, 10, 1),
                                                (5, 8, 3, 4, 1), (36, 4, 1, 13, 1)])
def test_adjoint_one_point_set(dtype, N, N_max, s, p, cross):
    """same-level lists (the plan is its own adjoint view) and cross-level lists (transposed lists): device vs oracle for a
    potential cotangent, a field cotangent and both; both kernel families; and the dot-product identity on the device alone."""
    pos, q = inputs.uniform_cube(N, 91, dtype)
    rng = np.random.default_rng(92)
    ubar, fbar = rng.standard_normal(N).astype(dtype), rng.standard_normal((N, 3)).astype(dtype)
    P = fmm.Plan(dev(pos), p, N_max, s, 0.77, cross_level=cross)
    Po = O.Plan(pos, p, N_max, s, 0.77, cross_level=cross)
    f32 = dtype == np.float32
    # the oracle forms every transposed translation column by column (K translates each): sizes are chosen for a few seconds per call
    cases = [(ubar, None), (None, fbar), (ubar, fbar)]
    wants = [Po.evaluate_adjoint(ub, fb, fp32_rule=f32) for ub, fb in cases]
    for variant in (0, 1):
        fmm.fmm_plan_set_m2l_variant(P.handle, variant)
        for (ub, fb), want in zip(cases, wants):
            got = P.evaluate_adjoint(dev(ub), dev(fb)).cpu().numpy()
            assert np.all(np.isfinite(got))
            assert rel2(got, want) <= TOL[dtype], (variant, ub is None, fb is None, rel2(got, want))
    fmm.fmm_plan_set_m2l_variant(P.handle, 0)
    u, f = P.evaluate(dev(q))
    u, f = u.double().cpu().numpy(), f.double().cpu().numpy()
    qbar = P.evaluate_adjoint(dev(ubar), dev(fbar)).double().cpu().numpy()
    lhs, rhs = ubar.astype(np.float64) @ u + np.sum(fbar.astype(np.float64) * f), qbar @ q.astype(np.float64)
    scale = np.abs(ubar) @ np.abs(u) + np.sum(np.abs(fbar * f))
    assert abs(lhs - rhs) <= (2e-6 if f32 else 1e-12) * scale, (lhs, rhs, scale)  # rounding level, far below the truncation error
    P.close()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("Ns,Nt,N_max,s,p", [(3000, 2000, 32, 2, 6), (1024, 4096, 16, 3, 6), (700, 5000, 20, 1, 4), (300, 300, 8, 3, 8)])
def test_adjoint_separate_targets(dtype, Ns, Nt, N_max, s, p):
    sp, q = inputs.uniform_cube(Ns, 93, dtype)
    tp = (np.random.default_rng(94).random((Nt, 3)) * 1.6 - 0.3).astype(dtype)
    rng = np.random.default_rng(95)
    ubar, fbar = rng.standard_normal(Nt).astype(dtype), rng.standard_normal((Nt, 3)).astype(dtype)
    P = fmm.PlanTargets(dev(sp), dev(tp), p, N_max, s)
    Po = O.PlanST(sp, tp, p, N_max, s)
    f32 = dtype == np.float32
    for ub, fb in ((ubar, None), (None, fbar), (ubar, fbar)):
        got = P.evaluate_adjoint(dev(ub), dev(fb)).cpu().numpy()
        want = Po.evaluate_adjoint(ub, fb, fp32_rule=f32)
        assert rel2(got, want) <= TOL[dtype], (ub is None, fb is None, rel2(got, want))
    # forward evaluates still work after the adjoint (the view borrows the plan's coefficient arrays) and the identity holds
    u, f = P.evaluate(dev(q))
    uo, fo = Po.evaluate(q, fp32_rule=f32)
    assert rel2(u.cpu().numpy(), uo) <= TOL[dtype] and rel2(f.cpu().numpy(), fo) <= TOL[dtype]
    u, f = u.double().cpu().numpy(), f.double().cpu().numpy()
    qbar = P.evaluate_adjoint(dev(ubar), dev(fbar)).double().cpu().numpy()
    lhs, rhs = ubar.astype(np.float64) @ u + np.sum(fbar.astype(np.float64) * f), qbar @ q.astype(np.float64)
    assert abs(lhs - rhs) <= (2e-6 if f32 else 1e-12) * (np.abs(ubar) @ np.abs(u) + np.sum(np.abs(fbar * f)))
    P.close()


def test_adjoint_against_the_transposed_definition():
    """A^T ubar is the plain definition with sources and targets exchanged (orc_direct_st); error of the order of the forward one"""
    rng = np.random.default_rng(80)
    src = rng.random((3000, 3))
    tgt = rng.random((2000, 3)) * 1.6 - 0.3
    g = rng.uniform(-1, 1, 2000)
    P = fmm.PlanTargets(dev(src), dev(tgt), 10, 32, 2)
    got = P.evaluate_adjoint(dev(g), None).cpu().numpy()
    want, _ = O.direct_st(tgt, g, src)
    assert rel2(got, want) < 1e-4
    with pytest.raises(ValueError):
        P.evaluate_adjoint(None, None)
    with pytest.raises(ValueError):
        P.evaluate_adjoint(dev(g[:100]), None)  # wrong length: rejected by the binding before it reaches the library
    P.close()


def test_active_shielding_demo():
    """128 shield charges on a sphere of radius 2 are optimised by gradient descent so that the potential of 256
    random external charges (radius 5) has minimal variance on 1024 points at radius 1.5, while the shield's own potential at 1024
    points at radius 2.5 stays small (eqs. (16)-(19), w_in = 1, w_out = 0.2, w_reg = 0.1).  Loss and gradient come from fmm_evaluate
    and fmm_evaluate_adjoint only; the optimum of the quadratic problem from dense matrices of the definition is the yardstick."""
    rng = np.random.default_rng(81)
    sh, p_in, p_out = fib_sphere(128, 2.0), fib_sphere(1024, 1.5), fib_sphere(1024, 2.5)
    v = rng.normal(size=(256, 3))
    ext = np.ascontiguousarray(5.0 * v / np.linalg.norm(v, axis=1, keepdims=True))
    q_ext = rng.uniform(-1, 1, 256)
    w_in, w_out, w_reg = 1.0, 0.2, 0.1
    P_in = fmm.PlanTargets(dev(sh), dev(p_in), 8, 32, 2)
    P_out = fmm.PlanTargets(dev(sh), dev(p_out), 8, 32, 2)
    P_ext = fmm.PlanTargets(dev(ext), dev(p_in), 8, 32, 2)
    phi_ext_in = P_ext.evaluate(dev(q_ext), want_field=False)[0]

    def loss_and_grad(q):
        tq = dev(q)
        a = phi_ext_in + P_in.evaluate(tq, want_field=False)[0]
        c = a - a.mean()                                  # eq. (16)
        b = P_out.evaluate(tq, want_field=False)[0]        # eq. (17)
        L = w_in * float(c @ c) + w_out * float(b @ b) + w_reg * float(q @ q)
        # d/dq: the centring projector is symmetric and idempotent, so grad = 2 w_in A_in^T c + 2 w_out A_out^T b + 2 w_reg q
        g = 2 * w_in * P_in.evaluate_adjoint(c.contiguous(), None) + 2 * w_out * P_out.evaluate_adjoint(b.contiguous(), None)
        return L, g.cpu().numpy() + 2 * w_reg * q

    def dense(src, tgt):
        return -1.0 / (4 * np.pi * np.linalg.norm(tgt[:, None, :] - src[None, :, :], axis=2))
    A_in, A_out = dense(sh, p_in), dense(sh, p_out)
    C = np.eye(1024) - np.ones((1024, 1024)) / 1024
    H = w_in * A_in.T @ C @ A_in + w_out * A_out.T @ A_out + w_reg * np.eye(128)
    q_star = np.linalg.solve(H, -w_in * A_in.T @ C @ (dense(ext, p_in) @ q_ext))
    L_star = loss_and_grad(q_star)[0]

    q = np.zeros(128)
    L0, g = loss_and_grad(q)
    g_ref = 2 * w_in * A_in.T @ C @ (dense(ext, p_in) @ q_ext)
    assert np.linalg.norm(g - g_ref) / np.linalg.norm(g_ref) < 1e-3
    step = 1.0 / (2 * np.linalg.eigvalsh(H)[-1])  # 1 / Lipschitz constant of the gradient
    losses = [L0]
    for _ in range(300):
        q = q - step * g
        L, g = loss_and_grad(q)
        losses.append(L)
    assert all(b <= a * (1 + 1e-6) for a, b in zip(losses, losses[1:]))  # "a simple gradient descent scheme suffices"
    assert losses[-1] < 0.5 * L0
    assert losses[-1] - L_star < 0.05 * (L0 - L_star), (L0, losses[-1], L_star)
    for P in (P_in, P_out, P_ext):
        P.close()
