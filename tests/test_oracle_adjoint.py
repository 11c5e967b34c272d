"""Pins for the oracle's adjoint evaluate (the gradient of a loss with respect to the charges; the evaluate is
linear in q, so the vector-Jacobian product is the transposed operator).  The adjoint is pinned against things other than itself:
the forward oracle (already pinned against the definition) through the dot-product identity, which a transposition must satisfy
to ROUND-OFF, not to truncation level; and the plain definition with sources and targets exchanged (orc_direct_st), which it must
approach like the forward evaluate does."""
import numpy as np
import pytest

from oracle import api as O
from paper_2511_15269_b200 import inputs


def rel2(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("N,N_max,s,p,cross", [(1500, 16, 2, 5, 0), (1500, 16, 2, 5, 1), (700, 8, 3, 3, 1), (300, 4, 1, 6, 0), (5, 8, 3, 4, 0), (40, 1, 2, 2, 1)])
def test_dot_product_identity_to_round_off(N, N_max, s, p, cross):
    """<ubar, A q> + <fbar, F q> == <A^T ubar + F^T fbar, q> for the FMM operators themselves (same lists, same order p):
    holds to rounding for an exact transposition, whatever the truncation error of A is.  Cross-level lists are not symmetric."""
    pos, q = inputs.uniform_cube(N, 71)
    rng = np.random.default_rng(72)
    ubar, fbar = rng.standard_normal(N), rng.standard_normal((N, 3))
    P = O.Plan(pos, p, N_max, s, 0.77, cross_level=cross)
    u, f = P.evaluate(q)
    for ub, fb in ((ubar, None), (None, fbar), (ubar, fbar)):
        qbar = P.evaluate_adjoint(ub, fb)
        lhs = (0.0 if ub is None else ub @ u) + (0.0 if fb is None else np.sum(fb * f))
        rhs = qbar @ q
        scale = (0.0 if ub is None else np.abs(ub) @ np.abs(u)) + (0.0 if fb is None else np.sum(np.abs(fb * f)))
        assert abs(lhs - rhs) < 1e-13 * scale, (lhs, rhs)


@pytest.mark.parametrize("Ns,Nt,N_max,s,p", [(900, 1400, 12, 2, 5), (1200, 300, 8, 3, 4), (64, 700, 4, 1, 6)])
def test_dot_product_identity_separate_targets(Ns, Nt, N_max, s, p):
    sp, q = inputs.uniform_cube(Ns, 73)
    tp = np.random.default_rng(74).random((Nt, 3)) * 1.6 - 0.3
    rng = np.random.default_rng(75)
    ubar, fbar = rng.standard_normal(Nt), rng.standard_normal((Nt, 3))
    P = O.PlanST(sp, tp, p, N_max, s, 0.77)
    u, f = P.evaluate(q)
    qbar = P.evaluate_adjoint(ubar, fbar)
    lhs, rhs = ubar @ u + np.sum(fbar * f), qbar @ q
    assert abs(lhs - rhs) < 1e-13 * (np.abs(ubar) @ np.abs(u) + np.sum(np.abs(fbar * f)))


def test_adjoint_approaches_the_transposed_definition():
    """A_ij = -1/(4 pi |t_i - s_j|): A^T ubar is the plain definition with the roles of sources and targets exchanged
    (orc_direct_st with "charges" ubar at the targets, evaluated at the sources); the error must fall with p like the forward one.
    The field part: column j of F is the field of a unit charge at s_j, taken from orc_direct_st as well."""
    sp, q = inputs.uniform_cube(400, 76)
    tp = np.random.default_rng(77).random((500, 3)) * 1.4 - 0.2
    rng = np.random.default_rng(78)
    ubar, fbar = rng.standard_normal(500), rng.standard_normal((500, 3))
    want_u, _ = O.direct_st(tp, ubar, sp)  # (A^T ubar)_j = -(1/4pi) sum_i ubar_i / |s_j - t_i|
    cols = [11, 200, 399]
    want_f = []
    for j in cols:
        e = np.zeros(400)
        e[j] = 1.0
        _, fj = O.direct_st(sp, e, tp)  # field at every target of a unit charge at s_j = column j of F
        want_f.append(np.sum(fbar * fj))
    errs = []
    for p in (2, 4, 6):
        P = O.PlanST(sp, tp, p, 8, 2, 0.77)
        errs.append((rel2(P.evaluate_adjoint(ubar, None), want_u),
                     max(abs(P.evaluate_adjoint(None, fbar)[j] - w) / abs(w) for j, w in zip(cols, want_f))))
    for a, b in zip(errs, errs[1:]):
        assert b[0] < 0.5 * a[0], errs
    assert errs[-1][0] < 2e-3 and errs[-1][1] < 2e-2, errs
    assert errs[-1][1] < 0.3 * errs[0][1], errs


def test_single_set_same_level_operator_is_symmetric():
    """One point set, same-level lists: the lists are symmetric and M2M^T = L2L, M2L(t<-s)^T = M2L(s<-t), P2M^T = L2P, so the
    FMM potential operator equals its own transpose up to rounding -- the adjoint of ubar is the forward potential of q = ubar."""
    pos, _ = inputs.uniform_cube(1200, 79)
    ubar = np.random.default_rng(80).standard_normal(1200)
    P = O.Plan(pos, 6, 16, 2, 0.77)
    u, _ = P.evaluate(ubar)
    assert rel2(P.evaluate_adjoint(ubar, None), u) < 1e-12
