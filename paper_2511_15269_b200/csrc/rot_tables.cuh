// rot_tables.cuh -- compile-time operator tables of the register ("fast") translation kernels (xlate_fast.cu).
//
// Same normalised representation as tables.cu (which builds the run-time copies in long double for the generic
// kernels); here every entry is a constant expression, so that after full unrolling each matrix entry becomes an
// immediate operand of an FFMA and structural zeros cost nothing.
//
//   B_n (2n+1)x(2n+1), row-major at boff(n): polar rotation of degree n, Q_n(theta) = B_n Z_n(theta) B_n^T with
//       B_n = Z_n(pi/2) Q_n(pi/2)  (a rotation about y is a rotation about z conjugated by a fixed quarter turn; this
//       replaces the on-the-fly Wigner-d recursion of PAPER.md:154 / App. B.2).  Three quarters of
//       the entries vanish (cos/sin-type decoupling and the parity d^n_{m',-m}(pi/2) = (-1)^(n+m') d^n_{m',m}(pi/2)).
//   Q_n = the normalised real-basis polar rotation by pi/2 itself.  Because Q_n^T = Z_n(pi) Q_n Z_n(pi) (a rotation by -pi/2
//       about y is the rotation by +pi/2 conjugated by a half turn about z), B_n^T = Z(pi) Q_n Z(pi/2) and therefore
//           B Z(theta) B^T = Z(pi/2) Q Z(theta + pi) Q Z(pi/2):
//       ONE constant matrix applied twice between azimuthal rotations.  The register kernels use this form, which lets the
//       forward and the inverse rotation of a translation share one copy of the Q code and one copy of the Z code in a
//       run-time loop (xlate_reg.cuh translate_qz) -- the whole kernel then fits the 32 KB instruction cache of an SM.
//   H[m][n][k] = (-1)^(k+m) (n+k)! / sqrt((n-m)!(n+m)!(k-m)!(k+m)!)          M2L z-shift, App. B.3
//   A[m][n][k] = sqrt((n-m)!(n+m)! / ((k-m)!(k+m)!)) / (n-k)!,  k <= n         M2M; L2L uses A[m][k][n]
#pragma once

namespace fmm {
namespace ct {

constexpr int PF = 12;  // largest order with a register kernel
constexpr int PF1 = PF + 1;

constexpr int boff(int n) { return n * (2 * n - 1) * (2 * n + 1) / 3; }
constexpr int NB = boff(PF + 1);

constexpr double csqrt(double x) {
    if (x <= 0.0) return 0.0;
    double g = x > 1.0 ? x : 1.0;
    for (int i = 0; i < 200; ++i) {
        const double h = 0.5 * (g + x / g);
        if (h == g) break;
        g = h;
    }
    return g;
}

struct Fact {
    double f[2 * PF + 2];
};
constexpr Fact make_fact() {
    Fact F{};
    F.f[0] = 1.0;
    for (int i = 1; i < 2 * PF + 2; ++i) F.f[i] = F.f[i - 1] * (double)i;
    return F;
}
constexpr Fact kFact = make_fact();

constexpr double binom(int n, int k) { return (k < 0 || k > n) ? 0.0 : kFact.f[n] / (kFact.f[k] * kFact.f[n - k]); }

// Wigner small-d at pi/2 (textbook explicit sum with cos = sin = 2^-1/2), written with binomials:
// d^j_{mp,m}(pi/2) = 2^-j sqrt((j+mp)!(j-mp)!/((j+m)!(j-m)!)) sum_k (-1)^(k-m+mp) C(j+m,k) C(j-m,k-m+mp)
constexpr double dhalf(int j, int mp, int m) {
    double sum = 0.0;
    for (int k = 0; k <= j + m; ++k) {
        const int k2 = k - m + mp;
        if (k2 < 0 || k2 > j - m) continue;
        const double t = binom(j + m, k) * binom(j - m, k2);
        sum += (k2 % 2) ? -t : t;
    }
    double s = sum * csqrt(kFact.f[j + mp] * kFact.f[j - mp] / (kFact.f[j + m] * kFact.f[j - m]));
    for (int i = 0; i < j; ++i) s *= 0.5;
    return s;
}

struct RotTab {
    double B[NB];
    double Q[NB];  // Q_n = normalised polar rotation by pi/2 (same layout as B); Q_n^T = Z_n(pi) Q_n Z_n(pi)
    double H[PF1][PF1][PF1];
    double A[PF1][PF1][PF1];
};

constexpr RotTab make_rot_tab() {
    RotTab T{};
    const double sq2 = csqrt(2.0);
    for (int n = 0; n <= PF; ++n) {
        const int w = 2 * n + 1;
        double Q[(2 * PF + 1) * (2 * PF + 1)] = {};
        // normalised polar rotation at pi/2: cos-type block (m,k >= 0) and sin-type block (m,k < 0)
        for (int m = 0; m <= n; ++m)
            for (int k = 0; k <= n; ++k) {
                const double em = m == 0 ? 1.0 : sq2, ek = k == 0 ? 1.0 : sq2;
                double v = 0.0;
                if (k == 0) v = em * dhalf(n, m, 0);
                else v = em / ek * (dhalf(n, m, k) + ((k % 2) ? -1.0 : 1.0) * dhalf(n, m, -k));
                Q[(n + m) * w + (n + k)] = v;
            }
        for (int m = 1; m <= n; ++m)
            for (int k = 1; k <= n; ++k) Q[(n - m) * w + (n - k)] = dhalf(n, m, k) - ((k % 2) ? -1.0 : 1.0) * dhalf(n, m, -k);
        for (int i = 0; i < w * w; ++i) {
            double v = Q[(i / w) * w + (i % w)];
            if (v < 1e-13 && v > -1e-13) v = 0.0;  // structural zeros
            T.Q[boff(n) + i] = v;
        }
        // B = Z(pi/2) Q : row m of B = cos(m pi/2) Q[m] - sin(m pi/2) Q[-m]
        for (int m = -n; m <= n; ++m) {
            const int r4 = ((m % 4) + 4) % 4;
            const double c = (r4 == 0) ? 1.0 : (r4 == 2 ? -1.0 : 0.0);
            const double s = (r4 == 1) ? 1.0 : (r4 == 3 ? -1.0 : 0.0);
            for (int k = -n; k <= n; ++k) {
                double v = c * Q[(n + m) * w + (n + k)] - s * Q[(n - m) * w + (n + k)];
                if (v < 1e-13 && v > -1e-13) v = 0.0;  // structural zeros
                T.B[boff(n) + (n + m) * w + (n + k)] = v;
            }
        }
    }
    for (int m = 0; m <= PF; ++m)
        for (int n = m; n <= PF; ++n)
            for (int k = m; k <= PF; ++k) {
                const double den = csqrt(kFact.f[n - m] * kFact.f[n + m] * kFact.f[k - m] * kFact.f[k + m]);
                T.H[m][n][k] = (((k + m) % 2) ? -1.0 : 1.0) * kFact.f[n + k] / den;
                if (k <= n) T.A[m][n][k] = csqrt(kFact.f[n - m] * kFact.f[n + m] / (kFact.f[k - m] * kFact.f[k + m])) / kFact.f[n - k];
            }
    return T;
}

constexpr RotTab kTab = make_rot_tab();

// number of non-zero entries of B_0..B_p (MACs of one application of B or B^T at order p)
constexpr int bnnz(int p) {
    int c = 0;
    for (int n = 0; n <= p; ++n)
        for (int i = 0; i < (2 * n + 1) * (2 * n + 1); ++i) c += kTab.B[boff(n) + i] != 0.0;
    return c;
}

}  // namespace ct
}  // namespace fmm
