// xlate_reg.cuh -- building blocks of the register ("fast") translation kernels (xlate_fast.cu, m2l_packed.cu):
// compile-time loops, application of the constant matrices B_n / B_n^T of rot_tables.cuh with every entry an FFMA
// immediate, azimuthal rotations (App. B.1 PAPER.md:441 in the normalised basis) and cos/sin(m x) tables.
// translate_reg is the whole rotate / z-shift / rotate-back operator for one translation held in registers.
// The value type T is float, double, or the packed pair f2 (two independent translations per thread, f32x2 SASS).
#pragma once
#include <type_traits>
#include <utility>

#include "internal.cuh"
#include "rot_tables.cuh"

namespace fmm {
namespace xr {

// ---- packed pair of floats: lane-wise arithmetic on two independent translations (FADD2 / FMUL2 / FFMA2, sm_100)
struct f2 {
    unsigned long long v;
    f2() = default;
    __device__ __forceinline__ explicit f2(float x) { asm("mov.b64 %0, {%1, %1};" : "=l"(v) : "f"(x)); }
    __device__ __forceinline__ explicit f2(double x) : f2((float)x) {}
    __device__ __forceinline__ f2(float lo, float hi) { asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(lo), "f"(hi)); }
    __device__ __forceinline__ float lo() const { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return a; }
    __device__ __forceinline__ float hi() const { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return b; }
};
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { f2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2& operator*=(f2& a, f2 b) { a = a * b; return a; }
__device__ __forceinline__ f2 fma(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
// a*b - c   (ptxas contracts the packed form into one FFMA2 with a negated addend)
__device__ __forceinline__ f2 fmsub(f2 a, f2 b, f2 c) { return a * b - c; }
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

template <int n, bool TR>
constexpr double bent(int i, int j) {
    constexpr int w = 2 * n + 1;
    return TR ? ct::kTab.B[ct::boff(n) + j * w + i] : ct::kTab.B[ct::boff(n) + i * w + j];
}
template <int n, bool TR>
constexpr bool bfirst(int i, int j) {
    for (int jj = 0; jj < j; ++jj)
        if (bent<n, TR>(i, jj) != 0.0) return false;
    return true;
}

// v[o .. o+2n] <- B_n v  (TR = false)  or  B_n^T v  (TR = true)
template <typename T, int n, bool TR, int KV>
__device__ __forceinline__ void apply_B(T (&v)[KV]) {
    constexpr int w = 2 * n + 1, o = n * n;
    T t[w];
    sfor<w>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        T acc = T(0.f);
        sfor<w>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            constexpr double b = bent<n, TR>(i, j);
            if constexpr (b != 0.0) {
                if constexpr (bfirst<n, TR>(i, j)) acc = T(b) * v[o + j];
                else acc = fma(T(b), v[o + j], acc);
            }
        });
        t[i] = acc;
    });
    sfor<w>([&](auto ic) { v[o + decltype(ic)::value] = t[decltype(ic)::value]; });
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

// KIND 0 = M2M (b = child - parent), 1 = M2L (b = source - target), 2 = L2L (b = parent - child)   [DESIGN.md reading G3]
// v: input coefficients of the old centre (length scale a_old) -> output coefficients about the new centre (a_new).
// SYNC: the warps of a CTA meet at a barrier after every phase, so that they walk the (large, straight-line) code in
// lockstep and share instruction-cache lines.
template <typename T, int P, int KIND, bool SYNC, int KV>
__device__ __forceinline__ void translate_reg(T (&v)[KV], T bx, T by, T bz, T a_old, T a_new) {
    constexpr int P1 = P + 1;
    const T rxy2 = bx * bx + by * by;
    const T r2 = rxy2 + bz * bz;
    const T r = sqrt(r2), rxy = sqrt(rxy2);
    const T rinv = r > T(0) ? T(1) / r : T(0);
    const T rxyinv = rxy > T(0) ? T(1) / rxy : T(0);
    const T ct_ = r > T(0) ? bz * rinv : T(1), st_ = rxy * rinv;
    const T cp_ = rxy > T(0) ? bx * rxyinv : T(1), sp_ = by * rxyinv;
    T x1, x2;
    if constexpr (KIND == 0) { x1 = r / a_new; x2 = a_old / a_new; }
    else if constexpr (KIND == 1) { x1 = a_new * rinv; x2 = a_old * rinv; }
    else { x1 = -r / a_old; x2 = a_new / a_old; }

    T cph[P1], sph[P1], cth[P1], sth[P1];
    trig_table<T, P1>(cp_, sp_, cph, sph);
    trig_table<T, P1>(ct_, st_, cth, sth);

    // forward rotation, degree by degree; M2M / M2L fold the source scaling x2^k in
    {
        T pw = T(1);
        sfor<P>([&](auto nc) {
            constexpr int n = decltype(nc)::value + 1;
            if constexpr (KIND != 2) {
                pw *= x2;
                sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
            }
            apply_az<T, n, +1>(v, cph, sph);
            apply_B<T, n, true>(v);
            apply_az<T, n, +1>(v, cth, sth);
            apply_B<T, n, false>(v);
            if constexpr (SYNC && n >= 3) __syncthreads();
        });
    }

    // z-shift (App. B.3), order by order; only equal m couple
    if constexpr (KIND == 1) {
        sfor<2 * P + 1>([&](auto mi) {
            constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
            T t[cnt];
            sfor<cnt>([&](auto ni) {
                constexpr int n = am + decltype(ni)::value;
                constexpr double h0 = ct::kTab.H[am][n][am];
                T acc = T(h0) * v[am * am + am + m];
                sfor<cnt - 1>([&](auto ki) {
                    constexpr int k = am + 1 + decltype(ki)::value;
                    constexpr double h = ct::kTab.H[am][n][k];
                    acc = fma(T(h), v[k * k + k + m], acc);
                });
                t[decltype(ni)::value] = acc;
            });
            sfor<cnt>([&](auto ni) { v[(am + decltype(ni)::value) * (am + decltype(ni)::value + 1) + m] = t[decltype(ni)::value]; });
        });
        T pw = rinv;
        sfor<P1>([&](auto nc) {
            constexpr int n = decltype(nc)::value;
            sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
            pw *= x1;
        });
    } else {
        T pw1[P1];
        pw1[0] = T(1);
        sfor<P>([&](auto jc) { pw1[decltype(jc)::value + 1] = pw1[decltype(jc)::value] * x1; });
        if constexpr (KIND == 0) {
            // out[n] = sum_{k=|m|..n} A[|m|][n][k] x1^(n-k) v[k]   (v already scaled by x2^k): in place, n descending
            sfor<2 * P + 1>([&](auto mi) {
                constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
                sfor<cnt>([&](auto ni) {
                    constexpr int n = P - decltype(ni)::value;
                    T acc = v[n * n + n + m];  // A[m][n][n] = 1
                    sfor<n - am>([&](auto ki) {
                        constexpr int k = am + decltype(ki)::value;
                        constexpr double aa = ct::kTab.A[am][n][k];
                        acc = fma(T(aa) * pw1[n - k], v[k * k + k + m], acc);
                    });
                    v[n * n + n + m] = acc;
                });
            });
        } else {
            // out[n] = x2^n sum_{k=n..p} A[|m|][k][n] x1^(k-n) v[k]: in place, n ascending
            T pw2[P1];
            pw2[0] = T(1);
            sfor<P>([&](auto jc) { pw2[decltype(jc)::value + 1] = pw2[decltype(jc)::value] * x2; });
            sfor<2 * P + 1>([&](auto mi) {
                constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
                sfor<cnt>([&](auto ni) {
                    constexpr int n = am + decltype(ni)::value;
                    T acc = v[n * n + n + m];
                    sfor<P - n>([&](auto ki) {
                        constexpr int k = n + 1 + decltype(ki)::value;
                        constexpr double aa = ct::kTab.A[am][k][n];
                        acc = fma(T(aa) * pw1[k - n], v[k * k + k + m], acc);
                    });
                    v[n * n + n + m] = acc * pw2[n];
                });
            });
        }
    }

    // inverse rotation
    if constexpr (SYNC) __syncthreads();
    sfor<P>([&](auto nc) {
        constexpr int n = decltype(nc)::value + 1;
        apply_B<T, n, true>(v);
        apply_az<T, n, -1>(v, cth, sth);
        apply_B<T, n, false>(v);
        apply_az<T, n, -1>(v, cph, sph);
        if constexpr (SYNC && n >= 3) __syncthreads();
    });
}

}  // namespace xr
}  // namespace fmm
