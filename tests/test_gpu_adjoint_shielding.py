"""Gradient of a loss on the potential with respect to the charges ("Active Shielding").

The potential at targets t_i from charges at sources s_j is linear in q, phi = A q with A_ij = -1/(4 pi |t_i - s_j|), so the
vector-Jacobian product the paper obtains by JAX autodiff is q_bar = A^T phi_bar: the SAME kernel with the roles of sources and
targets exchanged.  On the device that is one more plan, fmm_plan_create_targets(sources = t, targets = s), evaluated on phi_bar.
It is the exact adjoint of the definition and agrees with the transpose of the forward FMM operator to truncation error (checked
below by the dot-product identity).  The cotangent of the FIELD output needs no new kernel either: field = -grad_t u, so
q_bar_j = sum_i f_bar_i . d field_i / d q_j = - sum_c [field component c, at s_j, of charges f_bar_c placed at the targets]: three
more evaluates of the role-swapped plan, one per component (test_field_adjoint_dot_product_identity).
The demo itself: 128 shield charges on a sphere of radius 2 are optimised by gradient descent so that the potential of
256 random external charges (radius 5) has minimal variance on 1024 points at radius 1.5, while the shield's own potential at
1024 points at radius 2.5 stays small (eqs. (16)-(19), w_in = 1, w_out = 0.2, w_reg = 0.1)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import api as O
from paper_2511_15269_b200 import fmm

pytestmark = pytest.mark.gpu


def fib_sphere(n, r):
    """n points spread evenly on a sphere of radius r (golden-angle spiral)"""
    k = np.arange(n) + 0.5
    z = 1.0 - 2.0 * k / n
    ph = np.pi * (1.0 + 5.0 ** 0.5) * k
    s = np.sqrt(1.0 - z * z)
    return np.ascontiguousarray(r * np.stack([s * np.cos(ph), s * np.sin(ph), z], axis=1))


class Op:
    """phi = A q at `tgt` from charges at `src` and its adjoint, both by the device FMM"""

    def __init__(self, src, tgt, p=8, N_max=32, s=2):
        ts, tt = torch.from_numpy(src).cuda(), torch.from_numpy(tgt).cuda()
        self.fwd = fmm.PlanTargets(ts, tt, p, N_max, s)
        self.adj = fmm.PlanTargets(tt, ts, p, N_max, s)  # roles exchanged

    def A(self, q):
        u, _ = self.fwd.evaluate(torch.from_numpy(np.ascontiguousarray(q)).cuda(), want_field=False)
        return u.cpu().numpy()

    def AT(self, g):
        u, _ = self.adj.evaluate(torch.from_numpy(np.ascontiguousarray(g)).cuda(), want_field=False)
        return u.cpu().numpy()

    def F(self, q):
        """field at tgt, (Nt, 3)"""
        _, f = self.fwd.evaluate(torch.from_numpy(np.ascontiguousarray(q)).cuda(), want_potential=False)
        return f.cpu().numpy()

    def FT(self, fbar):
        """adjoint of F: q_bar = -sum_c field_c of the charges fbar[:, c] at the targets, evaluated at the sources"""
        out = np.zeros(self.adj.Nt)
        for c in range(3):
            _, f = self.adj.evaluate(torch.from_numpy(np.ascontiguousarray(fbar[:, c])).cuda(), want_potential=False)
            out -= f.cpu().numpy()[:, c]
        return out


def test_adjoint_dot_product_identity():
    rng = np.random.default_rng(80)
    src = rng.random((3000, 3))
    tgt = rng.random((2000, 3)) * 1.6 - 0.3
    q, g = rng.uniform(-1, 1, 3000), rng.uniform(-1, 1, 2000)
    op = Op(src, tgt, p=10)
    lhs, rhs = float(g @ op.A(q)), float(op.AT(g) @ q)
    ud, _ = O.direct_st(src, q, tgt)
    exact = float(g @ ud)
    assert abs(lhs - exact) < 2e-4 * np.linalg.norm(g) * np.linalg.norm(ud)
    assert abs(rhs - exact) < 2e-4 * np.linalg.norm(g) * np.linalg.norm(ud)
    assert abs(lhs - rhs) < 2e-4 * np.linalg.norm(g) * np.linalg.norm(ud)
    # the adjoint plan against the plain definition of A^T g
    want, _ = O.direct_st(tgt, g, src)
    got = op.AT(g)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 1e-4


def test_field_adjoint_dot_product_identity():
    rng = np.random.default_rng(82)
    src = rng.random((2500, 3))
    tgt = rng.random((1800, 3)) * 1.6 - 0.3
    q, fbar = rng.uniform(-1, 1, 2500), rng.uniform(-1, 1, (1800, 3))
    op = Op(src, tgt, p=10)
    _, fd = O.direct_st(src, q, tgt)
    exact = float(np.sum(fbar * fd))
    scale = np.linalg.norm(fbar) * np.linalg.norm(fd)
    lhs, rhs = float(np.sum(fbar * op.F(q))), float(op.FT(fbar) @ q)
    assert abs(lhs - exact) < 5e-4 * scale and abs(rhs - exact) < 5e-4 * scale and abs(lhs - rhs) < 5e-4 * scale
    # against the plain definition of the transposed field operator: q_bar_j = -(1/4pi) sum_i fbar_i . (t_i - s_j) / |t_i - s_j|^3
    d = tgt[:, None, :] - src[None, :, :]
    r3 = np.linalg.norm(d, axis=2) ** 3
    want = -(np.einsum("ic,ijc->ij", fbar, d) / r3).sum(axis=0) / (4 * np.pi)
    got = op.FT(fbar)
    assert np.linalg.norm(got - want) / np.linalg.norm(want) < 1e-3


def test_active_shielding_demo():
    rng = np.random.default_rng(81)
    sh, p_in, p_out = fib_sphere(128, 2.0), fib_sphere(1024, 1.5), fib_sphere(1024, 2.5)
    v = rng.normal(size=(256, 3))
    ext = np.ascontiguousarray(5.0 * v / np.linalg.norm(v, axis=1, keepdims=True))
    q_ext = rng.uniform(-1, 1, 256)
    w_in, w_out, w_reg = 1.0, 0.2, 0.1
    op_in, op_out = Op(sh, p_in), Op(sh, p_out)
    phi_ext_in = Op(ext, p_in).A(q_ext)

    def loss_and_grad(q):
        a = phi_ext_in + op_in.A(q)
        c = a - a.mean()                      # eq. (16)
        b = op_out.A(q)                       # eq. (17)
        L = w_in * (c @ c) + w_out * (b @ b) + w_reg * (q @ q)
        # d/dq: the centring projector is symmetric and idempotent, so grad = 2 w_in A_in^T c + 2 w_out A_out^T b + 2 w_reg q
        return L, 2 * w_in * op_in.AT(c) + 2 * w_out * op_out.AT(b) + 2 * w_reg * q

    # reference optimum from the dense matrices of the definition (the loss is quadratic)
    def dense(src, tgt):
        return -1.0 / (4 * np.pi * np.linalg.norm(tgt[:, None, :] - src[None, :, :], axis=2))
    A_in, A_out = dense(sh, p_in), dense(sh, p_out)
    C = np.eye(1024) - np.ones((1024, 1024)) / 1024
    H = w_in * A_in.T @ C @ A_in + w_out * A_out.T @ A_out + w_reg * np.eye(128)
    q_star = np.linalg.solve(H, -w_in * A_in.T @ C @ (dense(ext, p_in) @ q_ext))
    L_star = loss_and_grad(q_star)[0]

    q = np.zeros(128)
    L0, g = loss_and_grad(q)
    # gradient against the dense definition at the start
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
