// xlate_reg.cuh -- building blocks of the register ("fast") translation kernels (xlate_fast.cu, xlate_smem.cuh):
// compile-time loops, application of the constant matrices Q_n of rot_tables.cuh with every entry an FFMA immediate (fp32) or a
// materialised constant shared by a symmetric pair (fp64), azimuthal rotations (App. B.1 PAPER.md:441 in the normalised basis) and
// cos/sin(m x) tables.
// translate_qz is the whole rotate / z-shift / rotate-back operator for one translation held in registers (the Q Z loop).
// The value type T is float or double.
#pragma once
#include <type_traits>
#include <utility>

#include "internal.cuh"
#include "rot_tables.cuh"

namespace fmm {
namespace xr {

// a*b - c and a*b + c in the value type
__device__ __forceinline__ float fmsub(float a, float b, float c) { return ::fmaf(a, b, -c); }
__device__ __forceinline__ double fmsub(double a, double b, double c) { return ::fma(a, b, -c); }
__device__ __forceinline__ float fma(float a, float b, float c) { return ::fmaf(a, b, c); }
__device__ __forceinline__ double fma(double a, double b, double c) { return ::fma(a, b, c); }

template <class F, int... I>
__device__ __forceinline__ void sfor_impl(F&& f, std::integer_sequence<int, I...>) {
    (f(std::integral_constant<int, I>{}), ...);
}
// compile-time loop: f(integral_constant<int, 0>) ... f(integral_constant<int, N-1>)
template <int N, class F>
__device__ __forceinline__ void sfor(F&& f) {
    if constexpr (N > 0) sfor_impl(f, std::make_integer_sequence<int, N>{});
}

// azimuthal rotation of degree n (App. B.1 PAPER.md:441 in the normalised basis); SG = +1 forward, -1 inverse
template <typename T, int n, int SG, int KV, int P1>
__device__ __forceinline__ void apply_az(T (&v)[KV], const T (&c)[P1], const T (&s)[P1]) {
    constexpr int o = n * n + n;
    sfor<n>([&](auto mc) {
        constexpr int m = decltype(mc)::value + 1;
        const T a = v[o + m], b = v[o - m];
        if constexpr (SG > 0) {
            v[o + m] = fmsub(a, c[m], b * s[m]);
            v[o - m] = fma(b, c[m], a * s[m]);
        } else {
            v[o + m] = fma(a, c[m], b * s[m]);
            v[o - m] = fmsub(b, c[m], a * s[m]);
        }
    });
}

// cos(m x), sin(m x), m = 0..P, from cos x, sin x by the addition theorem
template <typename T, int P1>
__device__ __forceinline__ void trig_table(T c1, T s1, T (&c)[P1], T (&s)[P1]) {
    c[0] = T(1.f);
    s[0] = T(0.f);
    sfor<P1 - 1>([&](auto mc) {
        constexpr int m = decltype(mc)::value + 1;
        c[m] = fmsub(c[m - 1], c1, s[m - 1] * s1);
        s[m] = fma(s[m - 1], c1, c[m - 1] * s1);
    });
}

// ------------------------------------------------------------------------------------------------------------------------
// The translation operator in "Q Z loop" form.  KIND 0 = M2M (b = child - parent), 1 = M2L (b = source - target),
// 2 = L2L (b = parent - child) [DESIGN.md reading G3]; v: coefficients about the old centre (length scale a_old) -> coefficients
// about the new centre (a_new).  With Q_n the (constant) polar rotation by pi/2 and Q_n^T = Z(pi) Q_n Z(pi)
// (rot_tables.cuh), B Z(theta) B^T = Z(pi/2) Q Z(theta + pi) Q Z(pi/2), so that one translation is
//     Z(pi/2 - phi) Q Z(pi - theta) Q  [ Z(pi/2) S Z(pi/2) ]  Q Z(theta + pi) Q Z(phi + pi/2),
// S = z-shift.  S acts on the orders +m and -m alike, hence commutes with the azimuthal rotations and
// Z(pi/2) S Z(pi/2) = Z(pi) S = (-1)^m S: a sign that is folded into the shift constants.  What is left is the sequence
//     Z  Q Z  Q S  Q Z  Q Z
// i.e. five trips of a RUN-TIME loop whose body holds ONE copy of the Q code (bnnz(p) FMAs), one copy of the azimuthal
// code and one copy of the shift.  The straight-line form (round 1) needs four copies of the constant-matrix code and four of
// the azimuthal code (35 KB of SASS at p = 8, 48 KB with prologue and epilogue); this form is 20 KB, so the whole kernel
// stays inside the 32 KB instruction cache of an SM.  Measured on B200 with a synthetic FFMA stream (4 warps per
// scheduler): bodies up to 32 KB issue at 0.97 instructions per clock and scheduler, bodies of 48 KB and more at 0.5.
// Matrix entries are immediates of the FMA that uses them (fp32) or are materialised by two uniform moves (fp64).  Measured on B200
// (N = 1M, fp64 M2L): entries from a compact __constant__ table in the order of use (one 16-byte uniform load per two entries)
// 1.89 vs 1.55 ms at p = 8 and 13.4 vs 11.3 ms at p = 12; entries from a table in shared memory (broadcast LDS.128, one per two
// entries) 1.87 vs 1.55 ms and 13.1 vs 11.3 ms: every memory-sourced operand loses against the two uniform moves.
template <typename T, int n, int i, int j>
__device__ __forceinline__ T q_coef() {
    constexpr double v = ct::kTab.Q[ct::boff(n) + i * (2 * n + 1) + j];
    return T(v);
}
// sg * H[am][n][k] / sg * A[am][n][k] with sg = +-1 (the sign is an operand modifier of the instruction that uses it)
template <typename T, int am, int n, int k, bool NEG>
__device__ __forceinline__ T h_coef() {
    constexpr double v = NEG ? -ct::kTab.H[am][n][k] : ct::kTab.H[am][n][k];
    return T(v);
}
template <typename T, int am, int n, int k, bool NEG>
__device__ __forceinline__ T a_coef() {
    constexpr double v = NEG ? -ct::kTab.A[am][n][k] : ct::kTab.A[am][n][k];
    return T(v);
}

template <int n>
constexpr double qent(int i, int j) {
    return ct::kTab.Q[ct::boff(n) + i * (2 * n + 1) + j];
}
template <int n>
constexpr bool qfirst(int i, int j) {
    for (int jj = 0; jj < j; ++jj)
        if (qent<n>(i, jj) != 0.0) return false;
    return true;
}

// dst[od .. od+2n] <- Q_n src[os .. os+2n]   (src and dst must be different register sets)                        FORM 0
// fp64 (FORM 1 / 2): a double is not an immediate but two uniform moves per use.  Q_n^T = D Q_n D with D = Z(pi) = diag((-1)^m)
// (rot_tables.cuh), hence Q D and D Q are SYMMETRIC matrices: FORM 1 applies S = Q D, FORM 2 applies S = D Q, and the entries (i, j) and
// (j, i) are served by ONE materialised constant -- half the moves, a quarter of all instructions of an fp64 translation.  The
// missing D costs nothing: next to an azimuthal rotation it is a half turn of the angle (Z(a) D = D Z(a) = Z(a + pi)), next to the
// z-shift it cancels the (-1)^m that the Q Z form folds into the shift constants.  fp32 entries are free immediates and keep the
// row-by-row form (shorter live ranges).
template <int n, int FORM>
constexpr double sent(int i, int j) {
    const double q = qent<n>(i, j);
    const int k = FORM == 1 ? j : i;  // the index whose order m = k - n carries the sign
    return FORM == 0 ? q : (((k - n) & 1) ? -q : q);
}
template <typename T, int n, int os, int od, int FORM = 0, int NS, int ND>
__device__ __forceinline__ void q_from_to(const T (&src)[NS], T (&dst)[ND]) {
    constexpr int w = 2 * n + 1;
    if constexpr (FORM != 0) {
        sfor<w>([&](auto ic) { dst[od + decltype(ic)::value] = T(0); });
        sfor<w>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            sfor<w - i>([&](auto dc) {
                constexpr int j = i + decltype(dc)::value;
                constexpr double b = sent<n, FORM>(i, j), bt = sent<n, FORM>(j, i);
                static_assert(b - bt < 1e-13 && bt - b < 1e-13, "Q D and D Q are symmetric");
                if constexpr (b != 0.0) {
                    const T c = T(b);
                    dst[od + i] = fma(c, src[os + j], dst[od + i]);
                    if constexpr (j != i) dst[od + j] = fma(c, src[os + i], dst[od + j]);
                }
            });
        });
    } else {
        sfor<w>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            T acc = T(0.f);
            sfor<w>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                constexpr double b = qent<n>(i, j);
                if constexpr (b != 0.0) {
                    if constexpr (qfirst<n>(i, j)) acc = q_coef<T, n, i, j>() * src[os + j];
                    else acc = fma(q_coef<T, n, i, j>(), src[os + j], acc);
                }
            });
            dst[od + i] = acc;
        });
    }
}
template <typename T>
constexpr int q_form(int which) { return sizeof(T) == 8 ? which : 0; }

// dst <- Z_n(angle) src for one degree (App. B.1 PAPER.md:441 in the normalised basis, forward sense); order 0 is copied
template <typename T, int n, int os, int od, int NS, int ND, int P1>
__device__ __forceinline__ void az_from_to(const T (&src)[NS], T (&dst)[ND], const T (&c)[P1], const T (&s)[P1]) {
    dst[od + n] = src[os + n];
    sfor<n>([&](auto mc) {
        constexpr int m = decltype(mc)::value + 1;
        const T a = src[os + n + m], b = src[os + n - m];
        dst[od + n + m] = fmsub(a, c[m], b * s[m]);
        dst[od + n - m] = fma(b, c[m], a * s[m]);
    });
}

// z-shift of App. B.3 in the normalised, scaled representation, times (-1)^m (see above); in place.
// M2L expects v already scaled by x2^k and applies x1^n / r; M2M expects v scaled by x2^k; L2L applies x2^n itself.
// SIGNED = false: the plain shift (the (-1)^m has been cancelled by the D of a symmetric Q form, see q_from_to)
template <typename T, int P, int KIND, bool FUSE, bool SIGNED = true, int KV>
__device__ __forceinline__ void shift_signed(T (&v)[KV], T x1, T x2, T rinv) {
    constexpr int P1 = P + 1;
    if constexpr (KIND == 1) {
        T pwo[P1];
        if constexpr (FUSE) {
            pwo[0] = rinv;
            sfor<P>([&](auto jc) { pwo[decltype(jc)::value + 1] = pwo[decltype(jc)::value] * x1; });
        }
        sfor<2 * P + 1>([&](auto mi) {
            constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
            [[maybe_unused]] constexpr double sg = (SIGNED && (am & 1)) ? -1.0 : 1.0;
            T t[cnt];
            if constexpr (!SIGNED) {
                // fp64 (symmetric forms): H[m][n][k] = (-1)^(k+m) X(n, k) with X symmetric; the caller has scaled v by (-x2)^k, so the
                // matrix left is (-1)^m X(n, k), and its entries (n, k) and (k, n) share one materialised constant (see q_from_to)
                sfor<cnt>([&](auto ni) { t[decltype(ni)::value] = T(0); });
                sfor<cnt>([&](auto ni) {
                    constexpr int n = am + decltype(ni)::value;
                    sfor<cnt - decltype(ni)::value>([&](auto dk) {
                        constexpr int k = n + decltype(dk)::value;
                        constexpr double b = ((k & 1) ? -1.0 : 1.0) * ct::kTab.H[am][n][k];
                        const T c = T(b);
                        t[n - am] = fma(c, v[k * k + k + m], t[n - am]);
                        if constexpr (k != n) t[k - am] = fma(c, v[n * n + n + m], t[k - am]);
                    });
                });
            } else {
                sfor<cnt>([&](auto ni) {
                    constexpr int n = am + decltype(ni)::value;
                    T acc = h_coef<T, am, n, am, (sg < 0)>() * v[am * am + am + m];
                    sfor<cnt - 1>([&](auto ki) {
                        constexpr int k = am + 1 + decltype(ki)::value;
                        acc = fma(h_coef<T, am, n, k, (sg < 0)>(), v[k * k + k + m], acc);
                    });
                    t[decltype(ni)::value] = acc;
                });
            }
            // the output scaling x1^n / r is also the write-back (no register copies inside the run-time loop of translate_qz)
            sfor<cnt>([&](auto ni) {
                constexpr int n = am + decltype(ni)::value;
                if constexpr (FUSE) v[n * n + n + m] = t[decltype(ni)::value] * pwo[n];
                else v[n * n + n + m] = t[decltype(ni)::value];
            });
        });
        if constexpr (!FUSE) {
            T pw = rinv;
            sfor<P1>([&](auto nc) {
                constexpr int n = decltype(nc)::value;
                sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
                pw *= x1;
            });
        }
    } else {
        T pw1[P1];
        pw1[0] = T(1);
        sfor<P>([&](auto jc) { pw1[decltype(jc)::value + 1] = pw1[decltype(jc)::value] * x1; });
        if constexpr (KIND == 0) {
            // out[n] = (-1)^m sum_{k=|m|..n} A[|m|][n][k] x1^(n-k) v[k]   (A[m][n][n] = 1): in place, n descending
            sfor<2 * P + 1>([&](auto mi) {
                constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
                [[maybe_unused]] constexpr double sg = (SIGNED && (am & 1)) ? -1.0 : 1.0;
                sfor<cnt>([&](auto ni) {
                    constexpr int n = P - decltype(ni)::value;
                    T acc = (SIGNED && (am & 1)) ? T(0) - v[n * n + n + m] : v[n * n + n + m];
                    sfor<n - am>([&](auto ki) {
                        constexpr int k = am + decltype(ki)::value;
                        acc = fma(a_coef<T, am, n, k, (sg < 0)>() * pw1[n - k], v[k * k + k + m], acc);
                    });
                    v[n * n + n + m] = acc;
                });
            });
        } else {
            // out[n] = (-1)^m x2^n sum_{k=n..p} A[|m|][k][n] x1^(k-n) v[k]: in place, n ascending
            T pw2[P1];
            pw2[0] = T(1);
            sfor<P>([&](auto jc) { pw2[decltype(jc)::value + 1] = pw2[decltype(jc)::value] * x2; });
            sfor<2 * P + 1>([&](auto mi) {
                constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
                [[maybe_unused]] constexpr double sg = (SIGNED && (am & 1)) ? -1.0 : 1.0;
                sfor<cnt>([&](auto ni) {
                    constexpr int n = am + decltype(ni)::value;
                    T acc = v[n * n + n + m];
                    sfor<P - n>([&](auto ki) {
                        constexpr int k = n + 1 + decltype(ki)::value;
                        acc = fma(a_coef<T, am, k, n, false>() * pw1[k - n], v[k * k + k + m], acc);
                    });
                    v[n * n + n + m] = acc * (T(sg) * pw2[n]);
                });
            });
        }
    }
}

// direction of b, scale ratios:  x1, x2 as in translate_reg
template <typename T, int KIND>
__device__ __forceinline__ void xlate_geometry(T bx, T by, T bz, T a_old, T a_new, T& ct_, T& st_, T& cp_, T& sp_, T& rinv, T& x1, T& x2) {
    const T rxy2 = bx * bx + by * by;
    const T r2 = rxy2 + bz * bz;
    const T r = sqrt(r2), rxy = sqrt(rxy2);
    rinv = r > T(0) ? T(1) / r : T(0);
    const T rxyinv = rxy > T(0) ? T(1) / rxy : T(0);
    ct_ = r > T(0) ? bz * rinv : T(1);
    st_ = rxy * rinv;
    cp_ = rxy > T(0) ? bx * rxyinv : T(1);
    sp_ = by * rxyinv;
    if constexpr (KIND == 0) { x1 = r / a_new; x2 = a_old / a_new; }
    else if constexpr (KIND == 1) { x1 = a_new * rinv; x2 = a_old * rinv; }
    else { x1 = -r / a_old; x2 = a_new / a_old; }
}

// Register copies would be real instructions inside a run-time loop (the state must sit in the same registers at every
// back edge), so Q never works in place: it is always paired with an azimuthal rotation that moves the degree between the state v
// and a per-degree temporary -- "A(alpha)": t = Z_n(alpha) v_n, v_n = Q_n t  and  "B(alpha)": t = Q_n v_n, v_n = Z_n(alpha) t.
// MODE 0: trips A(phi + pi/2), A(theta + pi), S, B(pi - theta), B(pi/2 - phi): no wasted work, two copies of the Q / Z code.
// MODE 1: trips A(phi + pi/2), A(theta + pi), S, A(0), A(pi - theta), Z(pi/2 - phi) in place: one copy of the Q code, one
//         identity rotation (2 p (p+1) extra FMAs).
template <typename T>
__device__ __forceinline__ void qz_angle(int k, T ct_, T st_, T cp_, T sp_, T& c1, T& s1) {
    // k: 0: phi + pi/2   1: theta + pi   2: pi - theta   3: pi/2 - phi   4: 0
    c1 = k == 0 ? T(0) - sp_ : (k == 3 ? sp_ : (k == 4 ? T(1) : T(0) - ct_));
    s1 = (k == 0 || k == 3) ? cp_ : (k == 1 ? T(0) - st_ : (k == 2 ? st_ : T(0)));
}

// translate_qz with the geometry of the translation given (xlate_geometry): cos / sin of the polar and azimuthal angle, 1/r, x1, x2
template <typename T, int P, int KIND, int MODE, int KV>
__device__ __forceinline__ void translate_qz_geo(T (&v)[KV], T ct_, T st_, T cp_, T sp_, T rinv, T x1, T x2);

template <typename T, int P, int KIND, int MODE, int KV>
__device__ __forceinline__ void translate_qz(T (&v)[KV], T bx, T by, T bz, T a_old, T a_new) {
    T ct_, st_, cp_, sp_, rinv, x1, x2;
    xlate_geometry<T, KIND>(bx, by, bz, a_old, a_new, ct_, st_, cp_, sp_, rinv, x1, x2);
    translate_qz_geo<T, P, KIND, MODE>(v, ct_, st_, cp_, sp_, rinv, x1, x2);
}

template <typename T, int P, int KIND, int MODE, int KV>
__device__ __forceinline__ void translate_qz_geo(T (&v)[KV], T ct_, T st_, T cp_, T sp_, T rinv, T x1, T x2) {
    constexpr int P1 = P + 1;
    if constexpr (KIND != 2) {  // M2M / M2L: the source scaling x2^n commutes with the rotations
        // fp64 M2L (symmetric shift, see shift_signed): (-x2)^n
        const T xs = (KIND == 1 && MODE == 2 && sizeof(T) == 8) ? T(0) - x2 : x2;
        T pw = T(1);
        sfor<P>([&](auto nc) {
            constexpr int n = decltype(nc)::value + 1;
            pw *= xs;
            sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
        });
    }
    if constexpr (MODE == 2) {  // Z | Q Z | Q S | Q Z | Q Z with Q in place (register copies at the back edge)
        // fp64: Q = D (D Q) with the symmetric D Q applied from paired constants (q_from_to FORM 2); the D that is left turns the
        // rotation that follows by pi -- Z(theta + pi) D = Z(theta), Z(pi - theta) D = Z(-theta), Z(pi/2 - phi) D = Z(3 pi/2 - phi)
        // -- and takes the (-1)^m out of the shift
        constexpr bool SYM = sizeof(T) == 8;
#pragma unroll 1
        for (int t = 0; t < 5; ++t) {
            if (t > 0)
                sfor<P>([&](auto nc) {
                    constexpr int n = decltype(nc)::value + 1;
                    T tt[2 * n + 1];
                    q_from_to<T, n, n * n, 0, q_form<T>(2)>(v, tt);
                    sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] = tt[decltype(ic)::value]; });
                });
            if (t == 2) {
                shift_signed<T, P, KIND, (MODE != 2), !SYM>(v, x1, x2, rinv);
            } else {
                T c1, s1, c[P1], s[P1];
                if constexpr (SYM) {
                    c1 = t == 0 ? T(0) - sp_ : (t == 4 ? T(0) - sp_ : ct_);
                    s1 = t == 0 ? cp_ : (t == 1 ? st_ : (t == 3 ? T(0) - st_ : T(0) - cp_));
                } else {
                    qz_angle<T>(t < 2 ? t : t - 1, ct_, st_, cp_, sp_, c1, s1);
                }
                trig_table<T, P1>(c1, s1, c, s);
                sfor<P>([&](auto nc) { apply_az<T, decltype(nc)::value + 1, +1>(v, c, s); });
            }
        }
        return;
    }
    constexpr int NT = MODE == 0 ? 5 : 6;
#pragma unroll 1
    for (int t = 0; t < NT; ++t) {
        if (t == 2) {
            shift_signed<T, P, KIND, (MODE != 2)>(v, x1, x2, rinv);
            continue;
        }
        T c1, s1, c[P1], s[P1];
        const int k = MODE == 0 ? (t < 2 ? t : t - 1) : (t < 2 ? t : (t == 3 ? 4 : t - 2));
        qz_angle<T>(k, ct_, st_, cp_, sp_, c1, s1);
        trig_table<T, P1>(c1, s1, c, s);
        if (MODE == 1 && t == 5) {
            sfor<P>([&](auto nc) { apply_az<T, decltype(nc)::value + 1, +1>(v, c, s); });
        } else if (MODE == 1 || t < 2) {
            sfor<P>([&](auto nc) {
                constexpr int n = decltype(nc)::value + 1;
                T tt[2 * n + 1];
                az_from_to<T, n, n * n, 0>(v, tt, c, s);
                q_from_to<T, n, 0, n * n>(tt, v);
            });
        } else {
            sfor<P>([&](auto nc) {
                constexpr int n = decltype(nc)::value + 1;
                T tt[2 * n + 1];
                q_from_to<T, n, n * n, 0>(v, tt);
                az_from_to<T, n, 0, n * n>(tt, v, c, s);
            });
        }
    }
}

}  // namespace xr
}  // namespace fmm
