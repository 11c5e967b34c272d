"""Pins for the oracle's Wigner-d, rotations (App. B.1-B.2) and z-shifts / composite translations
(App. B.3) against closed forms and exact identities -- none produced by the oracle."""
import math

import numpy as np
import pytest
from scipy.special import lpmv

from oracle import api as O

RNG = np.random.default_rng(123)


def _weights(p):
    return np.array([(1.0 if m == 0 else 2.0) * (1.0 if m >= 0 else -1.0) for n in range(p + 1) for m in range(-n, n + 1)])


def _p2m(p, pts, q, c):
    """eq. (13) PAPER.md:145"""
    return sum(qi * O.regular_basis(p, r - c) for r, qi in zip(pts, q))


def _p2l(p, pts, q, c):
    """exact local coefficients of far charges: D = sum q S^(r_i - c) (addition theorem, eq. (12) in the real basis)"""
    return sum(qi * O.singular_basis(p, r - c) for r, qi in zip(pts, q))


def _eval_local(p, D, x):
    """eq. (14) PAPER.md:148 without the -1/4pi"""
    return float(np.sum(_weights(p) * D * O.regular_basis(p, x)))


def _eval_multipole(p, C, x):
    return float(np.sum(_weights(p) * C * O.singular_basis(p, x)))


def Ry(a):
    return np.array([[math.cos(a), 0, math.sin(a)], [0, 1, 0], [-math.sin(a), 0, math.cos(a)]])


def Rz(a):
    return np.array([[math.cos(a), -math.sin(a), 0], [math.sin(a), math.cos(a), 0], [0, 0, 1]])


# ---------------------------------------------------------------- Wigner d (reading S6)
@pytest.mark.parametrize("beta", [0.3, 1.1, 2.7, -0.8, math.pi / 2])
def test_wigner_d_textbook_low_degree(beta):
    c, s = math.cos(beta), math.sin(beta)
    d = O.wigner_d
    assert abs(d(0, 0, 0, beta) - 1) < 1e-15
    # j=1 (standard table, z-y-z convention)
    assert abs(d(1, 1, 1, beta) - (1 + c) / 2) < 1e-15
    assert abs(d(1, 1, 0, beta) + s / math.sqrt(2)) < 1e-15
    assert abs(d(1, 1, -1, beta) - (1 - c) / 2) < 1e-15
    assert abs(d(1, 0, 0, beta) - c) < 1e-15
    assert abs(d(1, 0, 1, beta) - s / math.sqrt(2)) < 1e-15
    # j=2
    assert abs(d(2, 2, 2, beta) - (1 + c) ** 2 / 4) < 1e-15
    assert abs(d(2, 2, 1, beta) + (1 + c) * s / 2) < 1e-15
    assert abs(d(2, 2, 0, beta) - math.sqrt(6) / 4 * s * s) < 1e-15
    assert abs(d(2, 1, 0, beta) + math.sqrt(1.5) * s * c) < 1e-15
    assert abs(d(2, 0, 0, beta) - (3 * c * c - 1) / 2) < 1e-15
    assert abs(d(2, 1, 1, beta) - (2 * c * c + c - 1) / 2) < 1e-15
    assert abs(d(2, 1, -1, beta) - (-2 * c * c + c + 1) / 2) < 1e-15


@pytest.mark.parametrize("j", [3, 6, 10, 12, 14, 16])
def test_wigner_d_m0_column_is_associated_legendre(j):
    """d^j_{m,0}(b) = sqrt((j-m)!/(j+m)!) P_j^m(cos b) (P with Condon-Shortley phase).  Up to j = FMM_P_MAX = 16: the explicit
    sum (reading S6) cancels more and more digits with j; 1e-12 at j = 16 is still far inside the fp64 parity tolerance."""
    beta = 0.9
    for m in range(0, j + 1):
        want = math.sqrt(math.factorial(j - m) / math.factorial(j + m)) * lpmv(m, j, math.cos(beta))
        assert abs(O.wigner_d(j, m, 0, beta) - want) < (1e-13 if j <= 12 else 1e-12)


@pytest.mark.parametrize("j", [1, 4, 8, 12, 16])
def test_wigner_d_identity_orthogonality_symmetries(j):
    beta = 0.77
    ms = range(-j, j + 1)
    d = np.array([[O.wigner_d(j, a, b, beta) for b in ms] for a in ms])
    d0 = np.array([[O.wigner_d(j, a, b, 0.0) for b in ms] for a in ms])
    dm = np.array([[O.wigner_d(j, a, b, -beta) for b in ms] for a in ms])
    dpi = np.array([[O.wigner_d(j, a, b, math.pi) for b in ms] for a in ms])
    assert np.max(np.abs(d0 - np.eye(2 * j + 1))) < 1e-15
    assert np.max(np.abs(d @ d.T - np.eye(2 * j + 1))) < 1e-12
    assert np.max(np.abs(dm - d.T)) < 1e-13  # d(-b) = d(b)^T
    for a in ms:
        for b in ms:
            assert abs(d[a + j, b + j] - (-1) ** (a - b) * d[b + j, a + j]) < 1e-13
            assert abs(d[a + j, b + j] - d[-b + j, -a + j]) < 1e-13
            want = (-1) ** (j - b) if a == -b else 0.0
            assert abs(dpi[a + j, b + j] - want) < 1e-12  # S7: d(pi)
    # composition d(b1) d(b2) = d(b1+b2)
    d1 = np.array([[O.wigner_d(j, a, b, 0.3) for b in ms] for a in ms])
    d2 = np.array([[O.wigner_d(j, a, b, 0.47) for b in ms] for a in ms])
    assert np.max(np.abs(d1 @ d2 - d)) < 1e-12


# ---------------------------------------------------------------- rotations B.1 / B.2
def _cloud(n, scale, centre, rng=None):
    rng = RNG if rng is None else rng
    return centre + scale * (rng.random((n, 3)) - 0.5), rng.uniform(-1, 1, n)


@pytest.mark.parametrize("ang", [0.4, -1.3, 2.9])
def test_azimuthal_rotation_equals_recomputation(ang):
    """Reading G4: frame turns by +dphi == points moved by Rz(-dphi)."""
    p = 8
    pts, q = _cloud(7, 1.0, np.zeros(3))
    far = pts * 3 + np.array([4.0, 3.0, -5.0])
    moved, fmoved = pts @ Rz(-ang).T, far @ Rz(-ang).T
    C, D = _p2m(p, pts, q, 0), _p2l(p, far, q, 0)
    assert np.max(np.abs(O.rot_azimuthal(p, 0, C, ang) - _p2m(p, moved, q, 0))) < 1e-14
    assert np.max(np.abs(O.rot_azimuthal(p, 1, D, ang) - _p2l(p, fmoved, q, 0))) < 1e-13 * np.max(np.abs(D))


@pytest.mark.parametrize("ang", [0.4, -1.3, 2.9, math.pi])
def test_polar_rotation_equals_recomputation(ang):
    """Reading G2: frame turns by +dtheta == points moved by Ry(-dtheta); d_{n,k}^{|m|} = d^n_{m'=|m|,m=k}."""
    p = 8
    pts, q = _cloud(7, 1.0, np.zeros(3))
    far = pts * 3 + np.array([4.0, 3.0, -5.0])
    moved, fmoved = pts @ Ry(-ang).T, far @ Ry(-ang).T
    C, D = _p2m(p, pts, q, 0), _p2l(p, far, q, 0)
    assert np.max(np.abs(O.rot_polar(p, 0, C, ang) - _p2m(p, moved, q, 0))) < 1e-13
    Dn = np.array([math.factorial(n) for n in range(p + 1) for _ in range(2 * n + 1)]) / 5.0 ** np.array(
        [n + 1 for n in range(p + 1) for _ in range(2 * n + 1)])
    assert np.max(np.abs(O.rot_polar(p, 1, D, ang) - _p2l(p, fmoved, q, 0)) / Dn) < 1e-11


def test_polar_rotation_orthogonal_after_normalisation():
    """T W T^-1 orthogonal with T = diag(sqrt((n-|m|)!(n+|m|)!) * (sqrt2 if m != 0)); inverse = rotation by -b."""
    p, beta = 8, 1.234
    K = O.nk(p)
    W = np.array([O.rot_polar(p, 0, np.eye(K)[i], beta) for i in range(K)]).T
    Wl = np.array([O.rot_polar(p, 1, np.eye(K)[i], beta) for i in range(K)]).T
    Wm = np.array([O.rot_polar(p, 0, np.eye(K)[i], -beta) for i in range(K)]).T
    g = np.array([math.sqrt(math.factorial(n - abs(m)) * math.factorial(n + abs(m))) * (1.0 if m == 0 else math.sqrt(2.0))
                  for n in range(p + 1) for m in range(-n, n + 1)])
    Q = (g[:, None] * W) / g[None, :]
    assert np.max(np.abs(Q @ Q.T - np.eye(K))) < 1e-12
    assert np.max(np.abs(Wm @ W - np.eye(K))) < 1e-11
    # local-type rotation is the contragredient one: sum w D R^ is invariant
    w = _weights(p)
    assert np.max(np.abs((W.T * w[None, :]) @ Wl - np.diag(w))) < 1e-11
    # degrees and cos/sin types do not mix
    for i in range(K):
        for j in range(K):
            ni, nj = int(math.isqrt(i)), int(math.isqrt(j))
            mi, mj = i - ni * ni - ni, j - nj * nj - nj
            if ni != nj or (mi >= 0) != (mj >= 0):
                assert W[i, j] == 0.0


# ---------------------------------------------------------------- z shifts and composite translations (reading G3)
DIRS = [np.array(v, dtype=float) for v in [(0.3, -0.5, 0.7), (0, 0, 1.3), (0, 0, -0.9), (1.1, 0.4, 0), (-0.2, -0.9, -0.6), (0.0, 0.7, 0.0)]]


@pytest.mark.parametrize("p", [8, 16])
@pytest.mark.parametrize("b", DIRS)
def test_m2m_is_exact(b, p):
    """M2M(P2M about c_old; b = c_old - c_new) == P2M about c_new, to round-off, for all n <= p (p = 16 = FMM_P_MAX too)."""
    c_new = np.array([0.1, 0.2, -0.3])
    c_old = c_new + b
    pts, q = _cloud(9, 0.6, c_old)
    got = O.translate(O.M2M, p, _p2m(p, pts, q, c_old), b)
    want = _p2m(p, pts, q, c_new)
    assert np.max(np.abs(got - want)) < (1e-13 if p <= 8 else 2e-12) * max(1.0, np.max(np.abs(want)))
    # monopole only: C' = q R^(b)
    e0 = np.zeros(O.nk(p)); e0[0] = 2.5
    assert np.max(np.abs(O.translate(O.M2M, p, e0, b) - 2.5 * O.regular_basis(p, b))) < 1e-14


@pytest.mark.parametrize("p", [8, 16])
@pytest.mark.parametrize("b", DIRS)
def test_l2l_is_exact(b, p):
    """same polynomial before and after: sum w D R^(x - c_old) == sum w D' R^(x - c_new)."""
    c_new = np.array([0.1, 0.2, -0.3])
    c_old = c_new + b
    D = RNG.standard_normal(O.nk(p))
    Dn = O.translate(O.L2L, p, D, b)
    for x in (c_new + np.array([0.2, -0.1, 0.15]), c_new + np.array([-0.3, 0.25, 0.05])):
        a, bb = _eval_local(p, D, x - c_old), _eval_local(p, Dn, x - c_new)
        assert abs(a - bb) < (1e-12 if p <= 8 else 2e-11) * max(1.0, abs(a))


@pytest.mark.parametrize("p", [10, 16])
@pytest.mark.parametrize("b", DIRS)
def test_m2l_of_a_monopole_is_the_singular_basis(b, p):
    """A charge sitting exactly on c_s has C = (q,0,...); M2L must return D = q S^(c_s - c_t) exactly (no truncation)."""
    e0 = np.zeros(O.nk(p)); e0[0] = -1.7
    got = O.translate(O.M2L, p, e0, 3.0 * b)
    want = -1.7 * O.singular_basis(p, 3.0 * b)
    scale = np.array([math.factorial(n) / np.linalg.norm(3 * b) ** (n + 1) for n in range(p + 1) for _ in range(2 * n + 1)])
    # at p = 16 the explicit Wigner sum (reading S6) has lost about five digits for directions in the xy-plane (beta = pi/2)
    assert np.max(np.abs(got - want) / scale) < (1e-12 if p <= 10 else 5e-11)


@pytest.mark.parametrize("b", DIRS)
def test_m2l_converges_to_direct(b):
    c_t = np.array([0.1, 0.2, -0.3])
    c_s = c_t + 2.6 * b / np.linalg.norm(b)
    pts, q = _cloud(12, 1.0, c_s, np.random.default_rng(77))  # own generator: the pointwise decay check must not depend on test order
    x = c_t + np.array([0.15, -0.2, 0.1])
    exact = sum(qi / np.linalg.norm(x - r) for r, qi in zip(pts, q))
    errs = []
    for p in (2, 4, 6, 8, 10, 12):
        D = O.translate(O.M2L, p, _p2m(p, pts, q, c_s), c_s - c_t)
        errs.append(abs(_eval_local(p, D, x - c_t) - exact))
    assert errs[0] < 2e-2 and errs[3] < 2e-6 and errs[5] < 2e-8
    assert all(errs[i + 2] < errs[i] for i in range(4))  # geometric decay (pointwise, so compared two steps apart)
    # low-order coefficients converge to the exact local coefficients sum q S^(r_i - c_t)
    p = 14
    D = O.translate(O.M2L, p, _p2m(p, pts, q, c_s), c_s - c_t)
    Dex = _p2l(p, pts, q, c_t)
    assert np.max(np.abs(D[:9] - Dex[:9])) < 1e-6


def test_zshift_matches_composite_on_plus_z():
    p, r = 6, 1.7
    v = RNG.standard_normal(O.nk(p))
    for kind in (O.M2M, O.M2L, O.L2L):
        assert np.max(np.abs(O.shift(kind, p, v, r) - O.translate(kind, p, v, np.array([0, 0, r])))) < 1e-13


def test_multipole_evaluation_far_away_matches_direct():
    """monopole = total charge (R^_0^0 = 1) and sum w C S^(x - c) ~ direct, far from the sources."""
    p = 16
    c = np.array([0.5, 0.5, 0.5])
    pts, q = _cloud(20, 1.0, c)
    C = _p2m(p, pts, q, c)
    assert abs(C[0] - np.sum(q)) < 1e-14
    x = c + np.array([2.0, -2.2, 2.1])
    exact = sum(qi / np.linalg.norm(x - r) for r, qi in zip(pts, q))
    assert abs(_eval_multipole(p, C, x - c) - exact) < 1e-11 * abs(exact) + 1e-13
