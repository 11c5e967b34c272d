"""Pins for the oracle's basis functions (App. A) against closed forms.

None of these tests calls back into the oracle to produce its own expectation: expectations are the
associated-Legendre definitions (scipy.special.lpmv, Condon-Shortley phase, as PAPER.md:355),
finite differences, and the plain 1/|r-r'|.
"""
import math

import numpy as np
import pytest
from scipy.special import lpmv

from oracle import api as O


def _sph(r):
    x, y, z = r
    rr = math.sqrt(x * x + y * y + z * z)
    return rr, math.acos(z / rr), math.atan2(y, x)


def _closed_regular(p, r):
    """R_n^m = alpha r^n P_n^|m|(cos t) e^{i m phi}, alpha = (-1)^m/(n+|m|)!;
    real basis = Re for m>=0, Im(R_n^m) for m<0."""
    rr, th, ph = _sph(r)
    out = np.zeros(O.nk(p))
    for n in range(p + 1):
        for m in range(-n, n + 1):
            am = abs(m)
            c = (-1.0) ** am / math.factorial(n + am) * rr**n * lpmv(am, n, math.cos(th))
            out[O.idx(n, m)] = c * math.cos(m * ph) if m >= 0 else c * math.sin(m * ph)
    return out


def _closed_singular(p, r):
    """S_n^m = beta r^-(n+1) P_n^|m| e^{i m phi}, beta = (-1)^m (n-|m|)!;
    real basis = Re(S_n^m) for m>=0, Im(S_n^{|m|}) for m<0."""
    rr, th, ph = _sph(r)
    out = np.zeros(O.nk(p))
    for n in range(p + 1):
        for m in range(-n, n + 1):
            am = abs(m)
            c = (-1.0) ** am * math.factorial(n - am) * rr ** (-(n + 1)) * lpmv(am, n, math.cos(th))
            out[O.idx(n, m)] = c * math.cos(am * ph) if m >= 0 else c * math.sin(am * ph)
    return out


PTS = [np.array(v) for v in [(0.3, -0.2, 0.5), (-0.7, 0.1, -0.4), (0.05, 0.9, 0.2), (1.3, 1.1, -2.0), (0.0, 0.0, 0.8), (0.4, 0.0, 0.0)]]


@pytest.mark.parametrize("r", PTS)
def test_regular_basis_closed_form(r):
    p = 10
    got, want = O.regular_basis(p, r), _closed_regular(p, r)
    scale = np.array([np.linalg.norm(r) ** n / math.factorial(n) for n in range(p + 1) for _ in range(2 * n + 1)])
    assert np.max(np.abs(got - want) / scale) < 1e-12


@pytest.mark.parametrize("r", PTS)
def test_singular_basis_closed_form(r):
    p = 10
    got, want = O.singular_basis(p, r), _closed_singular(p, r)
    scale = np.array([math.factorial(n) * np.linalg.norm(r) ** (-(n + 1)) for n in range(p + 1) for _ in range(2 * n + 1)])
    assert np.max(np.abs(got - want) / scale) < 1e-12


def test_base_cases_printed_in_paper(golden_dir):
    vals = {}
    for line in open(golden_dir + "/paper_values.txt"):
        line = line.split("#")[0].split()
        if len(line) == 2:
            vals[line[0]] = float(line[1])
    r = np.array([0.37, -0.61, 0.22])
    R = O.regular_basis(1, r)
    G = O.regular_grad(1, r)
    assert R[O.idx(0, 0)] == 1.0
    assert R[O.idx(1, 1)] == vals["R11_over_x"] * r[0]
    assert R[O.idx(1, -1)] == vals["R1m1_over_y"] * r[1]
    assert R[O.idx(1, 0)] == r[2]
    assert G[O.idx(1, 1)].tolist() == [vals["gradR11_x"], 0.0, 0.0]
    assert G[O.idx(1, -1)].tolist() == [0.0, vals["gradR1m1_y"], 0.0]
    S = O.singular_basis(1, r)
    rr = np.linalg.norm(r)
    assert abs(S[O.idx(0, 0)] - 1 / rr) < 1e-15
    assert abs(S[O.idx(1, 1)] - r[0] / rr**3) < 1e-14
    assert abs(S[O.idx(1, -1)] - r[1] / rr**3) < 1e-14


@pytest.mark.parametrize("r", PTS[:4])
def test_regular_grad_finite_differences(r):
    """Reading G1: with the minus sign printed at PAPER.md:419 this fails with error ~0.4."""
    p, h = 8, 1e-5
    G = O.regular_grad(p, r)
    for c in range(3):
        e = np.zeros(3)
        e[c] = h
        fd = (O.regular_basis(p, r + e) - O.regular_basis(p, r - e)) / (2 * h)
        assert np.max(np.abs(G[:, c] - fd)) < 2e-9 * max(1.0, np.linalg.norm(r)) ** p


@pytest.mark.parametrize("r", PTS[:4])
def test_regular_grad_ladder_identities(r):
    """App. A.3 integrates to the ladder identities of the complex basis R_n^m = R^_n^m - i R^_n^-m,
    R_n^-m = (-1)^m conj R_n^m:  d/dz R_n^m = R_{n-1}^m,  (d/dx + i d/dy) R_n^m = -R_{n-1}^{m+1},
    (d/dx - i d/dy) R_n^m = R_{n-1}^{m-1}.  A second, independent pin of the oracle's grad R^ (a wrong sign or index in A.3
    breaks one of the three), and the identity the CUDA L2P kernel uses instead of the A.3 recursions."""
    p = 8
    R, G = O.regular_basis(p, r), O.regular_grad(p, r)

    def Rc(n, m):
        if abs(m) > n:
            return 0j
        if m >= 0:
            return R[O.idx(n, m)] - 1j * (R[O.idx(n, -m)] if m > 0 else 0.0)
        return (-1) ** m * np.conj(Rc(n, -m))

    def Gc(n, m, c):  # gradient component c of the complex R_n^m, m >= 0
        return G[O.idx(n, m), c] - 1j * (G[O.idx(n, -m), c] if m > 0 else 0.0)

    scale = max(1.0, np.linalg.norm(r)) ** p
    for n in range(1, p + 1):
        for m in range(0, n + 1):
            gx, gy, gz = Gc(n, m, 0), Gc(n, m, 1), Gc(n, m, 2)
            assert abs(gz - Rc(n - 1, m)) < 1e-12 * scale
            assert abs((gx + 1j * gy) + Rc(n - 1, m + 1)) < 1e-12 * scale
            assert abs((gx - 1j * gy) - Rc(n - 1, m - 1)) < 1e-12 * scale


def test_regular_is_harmonic_and_homogeneous():
    r = np.array([0.3, 0.4, -0.2])
    p, h = 6, 1e-3
    lap = -6 * O.regular_basis(p, r)
    for c in range(3):
        e = np.zeros(3)
        e[c] = h
        lap += O.regular_basis(p, r + e) + O.regular_basis(p, r - e)
    assert np.max(np.abs(lap / h**2)) < 1e-6
    R2 = O.regular_basis(p, 2 * r)
    R1 = O.regular_basis(p, r)
    for n in range(p + 1):
        for m in range(-n, n + 1):
            assert abs(R2[O.idx(n, m)] - 2.0**n * R1[O.idx(n, m)]) < 1e-14


def _weights(p):
    """(2 - delta_0m) sgn(m), eq. (14) PAPER.md:148 (sgn(0)=1)."""
    return np.array([(1.0 if m == 0 else 2.0) * (1.0 if m >= 0 else -1.0) for n in range(p + 1) for m in range(-n, n + 1)])


def test_addition_theorem_truncation_decay():
    """Reading G5: 1/|r - r'| = sum (2-d0m) sgn(m) R^(r_<) S^(r_>), error ~ (r_</r_>)^{p+1}."""
    rs = np.array([0.11, -0.07, 0.05])
    rb = np.array([0.6, 0.9, -0.5])
    exact = 1.0 / np.linalg.norm(rb - rs)
    ratio = np.linalg.norm(rs) / np.linalg.norm(rb)
    prev = None
    for p in (2, 4, 6, 8, 10, 12):
        approx = np.sum(_weights(p) * O.regular_basis(p, rs) * O.singular_basis(p, rb))
        err = abs(approx - exact) / exact
        assert err < 3.0 * ratio ** (p + 1)
        if prev is not None and prev > 1e-14:
            assert err < prev
        prev = err
    assert prev < 1e-11
