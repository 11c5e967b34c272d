// tables.cu -- constant tables of the normalised operators, generated on the host in extended precision
// and uploaded once per device (DeviceCtx).  Independent of oracle/ (different formulas: binomial form of d^n(pi/2)).
//
// Normalisation used by every kernel of the CUDA path:
//   regular functions   Rn_n^m(r) = g_n^m * R^_n^m(r),  g_n^m = sqrt((n-|m|)!(n+|m|)!) * (m != 0 ? sqrt2 : 1)
//   multipole of a box  M_n^m = sum_i q_i Rn_n^m((r_i - c)/a)               (a = box length scale)
//   local of a box      phi_far(r) = sum L_n^m Rn_n^m((r - c)/a)
// In this basis rotations are orthogonal and identical for M and L; the polar rotation by theta factors exactly as
//   Q_n(theta) = B_n Z_n(theta) B_n^T,   B_n = Z_n(pi/2) Q_n(pi/2)   (Z_n = azimuthal rotation),
// because a rotation about y is a rotation about z conjugated by a fixed quarter turn.  This replaces the
// on-the-fly Wigner-d recursion of PAPER.md:154 by constant, half-empty matrices B_n.
#include <cmath>
#include <map>
#include <mutex>

#include "internal.cuh"

namespace fmm {
namespace {

long double fact(int n) {
    long double f = 1.0L;
    for (int i = 2; i <= n; ++i) f *= (long double)i;
    return f;
}
long double binom(int n, int k) {
    if (k < 0 || k > n) return 0.0L;
    return fact(n) / (fact(k) * fact(n - k));
}
// d^j_{mp,m}(pi/2) = 2^-j sqrt((j+mp)!(j-mp)!/((j+m)!(j-m)!)) sum_k (-1)^(k+mp-m)... written with binomials:
// d^j_{mp,m}(b) = sum_k (-1)^(k-m+mp) sqrt((j+m)!(j-m)!(j+mp)!(j-mp)!)/((j+m-k)! k! (j-k-mp)! (k-m+mp)!) c^(2j-2k+m-mp) s^(2k-m+mp)
//              = sqrt((j+mp)!(j-mp)!/((j+m)!(j-m)!)) sum_k (-1)^(k-m+mp) C(j+m,k) C(j-m,k-m+mp) c^.. s^..
long double dhalf(int j, int mp, int m) {
    long double sum = 0.0L;
    for (int k = 0; k <= j + m; ++k) {
        const int k2 = k - m + mp;
        if (k2 < 0 || k2 > j - m) continue;
        const long double t = binom(j + m, k) * binom(j - m, k2);
        sum += ((k2 % 2) ? -t : t);
    }
    return sum * std::sqrt(fact(j + mp) * fact(j - mp) / (fact(j + m) * fact(j - m))) * std::pow(2.0L, -(long double)j);
}

void build(Tables& T) {
    {
        int nB = 0;
        for (int n = 0; n <= PMAX; ++n) nB += (2 * n + 1) * (2 * n + 1);
        std::vector<double> B(nB, 0.0);
        std::vector<float> Bf(nB, 0.f);
        for (int n = 0; n <= PMAX; ++n) {
            const int w = 2 * n + 1;
            std::vector<long double> Q((size_t)w * w, 0.0L);
            auto e = [](int m) { return m == 0 ? 1.0L : std::sqrt(2.0L); };
            // normalised polar rotation at pi/2: cos-type block (m,k >= 0), sin-type block (m,k < 0)
            for (int m = 0; m <= n; ++m)
                for (int k = 0; k <= n; ++k) {
                    long double v;
                    if (k == 0) v = e(m) * dhalf(n, m, 0);
                    else v = e(m) / e(k) * (dhalf(n, m, k) + ((k % 2) ? -1.0L : 1.0L) * dhalf(n, m, -k));
                    Q[(size_t)(n + m) * w + (n + k)] = v;
                }
            for (int m = 1; m <= n; ++m)
                for (int k = 1; k <= n; ++k)
                    Q[(size_t)(n - m) * w + (n - k)] = dhalf(n, m, k) - ((k % 2) ? -1.0L : 1.0L) * dhalf(n, m, -k);
            // B = Z(pi/2) Q : row m of B = cos(m pi/2) Q[m] - sin(m pi/2) Q[-m]
            double* Bn = B.data() + boff(n);
            for (int m = -n; m <= n; ++m) {
                const int r4 = ((m % 4) + 4) % 4;
                const long double c = (r4 == 0) ? 1.0L : (r4 == 2 ? -1.0L : 0.0L);
                const long double s = (r4 == 1) ? 1.0L : (r4 == 3 ? -1.0L : 0.0L);
                for (int k = -n; k <= n; ++k) {
                    long double v = c * Q[(size_t)(n + m) * w + (n + k)] - s * Q[(size_t)(n - m) * w + (n + k)];
                    if (std::fabs((double)v) < 1e-15) v = 0.0L;  // structural zeros
                    Bn[(n + m) * w + (n + k)] = (double)v;
                }
            }
        }
        for (int i = 0; i < nB; ++i) Bf[i] = (float)B[i];
        const int P1 = PMAX + 1;
        std::vector<double> H((size_t)P1 * P1 * P1, 0.0), A((size_t)P1 * P1 * P1, 0.0), g(KMAX, 0.0);
        for (int m = 0; m <= PMAX; ++m)
            for (int n = m; n <= PMAX; ++n)
                for (int k = m; k <= PMAX; ++k) {
                    const long double den = std::sqrt(fact(n - m) * fact(n + m) * fact(k - m) * fact(k + m));
                    H[((size_t)m * P1 + n) * P1 + k] = (double)((((k + m) % 2) ? -1.0L : 1.0L) * fact(n + k) / den);
                    if (k <= n)
                        A[((size_t)m * P1 + n) * P1 + k] =
                            (double)(std::sqrt(fact(n - m) * fact(n + m) / (fact(k - m) * fact(k + m))) / fact(n - k));
                }
        for (int n = 0; n <= PMAX; ++n)
            for (int m = -n; m <= n; ++m) {
                const int am = m < 0 ? -m : m;
                g[n * n + n + m] = (double)(std::sqrt(fact(n - am) * fact(n + am)) * (m ? std::sqrt(2.0L) : 1.0L));
            }
        T.h_B = B;
        FMM_CUDA_CHECK(cudaMalloc((void**)&T.d_B, nB * sizeof(double)));
        FMM_CUDA_CHECK(cudaMalloc((void**)&T.d_Bf, nB * sizeof(float)));
        FMM_CUDA_CHECK(cudaMalloc((void**)&T.d_H, H.size() * sizeof(double)));
        FMM_CUDA_CHECK(cudaMalloc((void**)&T.d_A, A.size() * sizeof(double)));
        FMM_CUDA_CHECK(cudaMalloc((void**)&T.d_g, g.size() * sizeof(double)));
        FMM_CUDA_CHECK(cudaMemcpy(T.d_B, B.data(), nB * sizeof(double), cudaMemcpyHostToDevice));
        FMM_CUDA_CHECK(cudaMemcpy(T.d_Bf, Bf.data(), nB * sizeof(float), cudaMemcpyHostToDevice));
        FMM_CUDA_CHECK(cudaMemcpy(T.d_H, H.data(), H.size() * sizeof(double), cudaMemcpyHostToDevice));
        FMM_CUDA_CHECK(cudaMemcpy(T.d_A, A.data(), A.size() * sizeof(double), cudaMemcpyHostToDevice));
        FMM_CUDA_CHECK(cudaMemcpy(T.d_g, g.data(), g.size() * sizeof(double), cudaMemcpyHostToDevice));
    }
}

std::mutex g_mu;
std::map<int, std::unique_ptr<DeviceCtx>> g_ctx;

}  // namespace

int current_device() {
    int dev = 0;
    FMM_CUDA_CHECK(cudaGetDevice(&dev));
    return dev;
}

DeviceCtx& device_ctx(int dev) {
    std::lock_guard<std::mutex> lock(g_mu);
    auto it = g_ctx.find(dev);
    if (it != g_ctx.end()) return *it->second;
    if (dev < 0 || dev >= MAX_DEVICES) { set_error("device ordinal out of range"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
    if (current_device() != dev) { set_error("device_ctx: not the current device"); throw CudaFail{FMM_ERR_INVALID_ARG}; }
    std::unique_ptr<DeviceCtx> c(new DeviceCtx());
    c->dev = dev;
    build(c->tab);  // throws on failure: nothing is cached then
    DeviceCtx& ref = *c;
    g_ctx[dev] = std::move(c);
    return ref;
}

}  // namespace fmm
