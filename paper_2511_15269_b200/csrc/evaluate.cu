// evaluate.cu -- the evaluate pipeline (stage order PAPER.md:251):
//   permute charges -> P2M (eq. 13) -> M2M (App. B) -> M2L (App. B) -> L2L -> L2P (eq. 14, App. A.3) -> P2P
// All coefficient arrays use the normalised, length-scaled representation described in tables.cu / DESIGN.md.
// This file holds the kernels that work for every order p <= FMM_P_MAX and both dtypes; the unrolled register
// translation kernels (M2M, M2L, L2L) live in xlate_fast.cu.
#include "internal.cuh"

namespace fmm {
namespace {

__constant__ double c_g[KMAX];   // g_n^m, double
__constant__ float c_gf[KMAX];   // g_n^m, float

template <typename T> struct V4;
template <> struct V4<float> { using type = float4; };
template <> struct V4<double> { using type = double4; };
template <typename T> __device__ inline typename V4<T>::type make4(T a, T b, T c, T d);
template <> __device__ inline float4 make4<float>(float a, float b, float c, float d) { return make_float4(a, b, c, d); }
template <> __device__ inline double4 make4<double>(double a, double b, double c, double d) { return make_double4(a, b, c, d); }

template <typename T> __device__ inline T gnorm(int idx);
template <> __device__ inline float gnorm<float>(int idx) { return c_gf[idx]; }
template <> __device__ inline double gnorm<double>(int idx) { return c_g[idx]; }

template <typename T> __device__ inline T rsqrt_t(T x);
template <> __device__ inline float rsqrt_t<float>(float x) { return rsqrtf(x); }
template <> __device__ inline double rsqrt_t<double>(double x) { return rsqrt(x); }

template <typename T> __device__ inline T r2_min();
template <> __device__ inline float r2_min<float>() { return 1.17549435e-38f; }  // FLT_MIN
template <> __device__ inline double r2_min<double>() { return 4.9406564584124654e-324; }  // any r^2 > 0

inline unsigned nblocks(int64_t n, int t) { return (unsigned)((n + t - 1) / t); }

// ------------------------------------------------------------------------------------------------ permute (a3)
template <typename T>
__global__ void permute_k(const T* __restrict__ pos_tree, const T* __restrict__ q, const int32_t* __restrict__ perm,
                          typename V4<T>::type* __restrict__ pq, const int32_t* __restrict__ src_slot, float* __restrict__ srcg, int64_t N) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const T x = pos_tree[3 * k], y = pos_tree[3 * k + 1], z = pos_tree[3 * k + 2], qq = q ? q[perm[k]] : T(0);  // q == nullptr: pure targets
    pq[k] = make4<T>(x, y, z, qq);
    if (srcg) {  // fp32 only: P2P source groups (-x[4], -y[4], -z[4], q[4]), see p2p_fast.cu
        const int32_t sl = src_slot[k];
        float* g = srcg + (int64_t)(sl >> 2) * 16 + (sl & 3);
        g[0] = -(float)x; g[4] = -(float)y; g[8] = -(float)z; g[12] = (float)qq;
    }
}

// ------------------------------------------------------------------------------------------------ basis recursions
// App. A.1 on scaled coordinates, degree by degree, two rotating degree slots indexed [n&1][m+P].
// emit(n, m, R^_n^m) is called for every (n,m), n ascending, with compile-time n, m after unrolling.
template <int P, typename T, typename F>
__device__ __forceinline__ void regular_rec(T x, T y, T z, F&& emit) {
    T R[2][2 * P + 1];
    const T r2 = x * x + y * y + z * z;
    R[0][P] = T(1);
    emit(0, 0, R[0][P]);
#pragma unroll
    for (int n = 1; n <= P; ++n) {
        const int c = n & 1, q = c ^ 1;
        // inner orders first (they read slot c = degree n-2 and slot q = degree n-1), then +-(n-1), then +-n
#pragma unroll
        for (int m = -(n - 2); m <= n - 2; ++m) {
            const int am = m < 0 ? -m : m;
            R[c][P + m] = (T(2 * n - 1) * z * R[q][P + m] - r2 * R[c][P + m]) * (T(1) / T((n - am) * (n + am)));
        }
        if (n == 1) {
            R[c][P] = z * R[q][P];
            R[c][P + 1] = x * T(0.5);
            R[c][P - 1] = -y * T(0.5);
        } else {
            const T dp = R[q][P + n - 1], dm = R[q][P - (n - 1)];
            R[c][P + n - 1] = z * dp;
            R[c][P - (n - 1)] = z * dm;
            R[c][P + n] = (x * dp + y * dm) * (T(1) / T(2 * n));
            R[c][P - n] = (x * dm - y * dp) * (T(1) / T(2 * n));
        }
#pragma unroll
        for (int m = -n; m <= n; ++m) emit(n, m, R[c][P + m]);
    }
}

// ------------------------------------------------------------------------------------------------ P2M (a4), warp per leaf
#ifndef FMM_WPB
#define FMM_WPB 4
#endif
constexpr int WARPS_PER_BLOCK = FMM_WPB;

// LPL = lanes per leaf: 32 (a warp per leaf) or 16 (two leaves per warp, for plans whose leaves hold <= 16 particles).
template <typename T, int P, int LPL>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) p2m_k(const typename V4<T>::type* __restrict__ pq, const int32_t* __restrict__ box_start,
                                                              const int32_t* __restrict__ box_count, const double* __restrict__ ctr,
                                                              const T* __restrict__ scale, int64_t leaf0, int64_t n_leaves, int Kp,
                                                              T* __restrict__ Mc) {
    constexpr int K = (P + 1) * (P + 1);
    constexpr int NJ = (K + 31) / 32;
    constexpr int LPW = 32 / LPL;  // leaves per warp
    const int lane = threadIdx.x & 31, hl = lane % LPL;
    const int64_t leaf = ((int64_t)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5)) * LPW + lane / LPL;
    const bool have = leaf < n_leaves;
    if (LPL == 32 && !have) return;
    const int64_t g = leaf0 + (have ? leaf : 0);
    const int st = box_start[g], cnt = have ? box_count[g] : 0;
    const double cx = ctr[3 * g], cy = ctr[3 * g + 1], cz = ctr[3 * g + 2];
    const T inva = T(1) / scale[g];
    if constexpr (NJ * 32 * sizeof(T) / 4 <= 128) {
        // every lane accumulates all K coefficients of its own particles in registers; one recursive-halving reduce-scatter
        // (K + K/2 + ... shuffles instead of 5 K) then leaves coefficients NJ*lane .. NJ*lane + NJ-1 on lane `lane`
        constexpr int KP = NJ * 32;
        T w[KP];
#pragma unroll
        for (int i = 0; i < KP; ++i) w[i] = T(0);
        const int cmax = LPL == 32 ? cnt : max(cnt, __shfl_xor_sync(0xffffffffu, cnt, 16));  // warp-uniform trip count
        for (int base = 0; base < cmax; base += LPL) {
            const int i = base + hl;
            T x = 0, y = 0, z = 0, q = 0;
            if (i < cnt) {
                const typename V4<T>::type v = pq[st + i];
                x = (T)((double)v.x - cx) * inva;
                y = (T)((double)v.y - cy) * inva;
                z = (T)((double)v.z - cz) * inva;
                q = v.w;
            }
            regular_rec<P, T>(x, y, z, [&](int n, int m, T val) { w[n * n + n + m] += q * val; });
        }
#pragma unroll
        for (int bit = LPL / 2, h = KP / 2; bit > 0; bit >>= 1, h >>= 1) {
            const bool up = (lane & bit) != 0;
#pragma unroll
            for (int i = 0; i < h; ++i) {
                const T send = up ? w[i] : w[i + h];
                const T keep = up ? w[i + h] : w[i];
                w[i] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
            }
        }
        constexpr int NF = KP / LPL;  // coefficients NF*hl .. NF*hl + NF-1 end up on lane hl of the leaf's lane group
#pragma unroll
        for (int j = 0; j < NF; ++j) {
            const int idx = NF * hl + j;
            if (have && idx < K) Mc[g * Kp + idx] = w[j] * gnorm<T>(idx);
        }
    } else {
        static_assert(LPL == 32 || NJ * 32 * sizeof(T) / 4 <= 128, "two leaves per warp need the register reduce-scatter path");
        T acc[NJ];
#pragma unroll
        for (int j = 0; j < NJ; ++j) acc[j] = T(0);
        for (int base = 0; base < cnt; base += 32) {
            const int i = base + lane;
            T x = 0, y = 0, z = 0, q = 0;
            if (i < cnt) {
                const typename V4<T>::type v = pq[st + i];
                x = (T)((double)v.x - cx) * inva;
                y = (T)((double)v.y - cy) * inva;
                z = (T)((double)v.z - cz) * inva;
                q = v.w;
            }
            regular_rec<P, T>(x, y, z, [&](int n, int m, T val) {
                const int idx = n * n + n + m;
                T v = q * val * gnorm<T>(idx);
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
                if (lane == (idx & 31)) acc[idx >> 5] += v;
            });
        }
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            const int idx = lane + 32 * j;
            if (idx < K) Mc[g * Kp + idx] = acc[j];
        }
    }
}

__device__ inline void idx_to_nm(int idx, int& n, int& m) {
    n = (int)sqrtf((float)idx);
    while (n * n > idx) --n;
    while ((n + 1) * (n + 1) <= idx) ++n;
    m = idx - n * n - n;
}

// ------------------------------------------------------------------------------------------------ L2P (a8) + finalize (a10), warp per leaf
template <typename T, int P, int LPL>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) l2p_k(const typename V4<T>::type* __restrict__ pq, const int32_t* __restrict__ box_start,
                                                              const int32_t* __restrict__ box_count, const double* __restrict__ ctr,
                                                              const T* __restrict__ scale, int64_t leaf0, int64_t n_leaves, int Kp,
                                                              const T* __restrict__ Lc, const typename V4<T>::type* __restrict__ near,
                                                              const int32_t* __restrict__ perm, T* __restrict__ pot, T* __restrict__ field) {
    constexpr int K = (P + 1) * (P + 1);
    constexpr int KD = P > 0 ? P * P : 1;  // coefficients of degree <= P-1
    // The field is evaluated from three DERIVED expansions instead of running the grad R^ recursions of App. A.3
    // per particle.  In the paper's basis (R_n^m = R^_n^m - i R^_n^-m, R_n^-m = (-1)^m conj R_n^m) the
    // recursions of A.3 integrate to the ladder identities
    //     d/dz R_n^m = R_{n-1}^m,   (d/dx + i d/dy) R_n^m = -R_{n-1}^{m+1},   (d/dx - i d/dy) R_n^m = R_{n-1}^{m-1}
    // (pinned against the finite differences of the oracle's A.3 in tests/test_oracle_basis.py), so that for weights w
    //     d/dx sum w_n^m R^_n^m = sum X_{n-1}^k R^_{n-1}^k   etc. with the two- and three-term formulas below.  Per particle
    // this leaves one R^ recursion and 4 FMAs per coefficient.
    constexpr int LPW = 32 / LPL;  // leaves per warp (LPL lanes per leaf, see p2m_k)
    __shared__ T sLs[WARPS_PER_BLOCK * LPW][K];
    __shared__ T sDs[WARPS_PER_BLOCK * LPW][3][KD];
    const int lane = threadIdx.x & 31, hl = lane % LPL, w = (threadIdx.x >> 5) * LPW + lane / LPL;
    const int64_t leaf = (int64_t)blockIdx.x * WARPS_PER_BLOCK * LPW + w;
    const bool have = leaf < n_leaves;
    if (LPL == 32 && !have) return;
    const int64_t g = leaf0 + (have ? leaf : 0);
    const int st = box_start[g], cnt = have ? box_count[g] : 0;
    const double cx = ctr[3 * g], cy = ctr[3 * g + 1], cz = ctr[3 * g + 2];
    const T inva = T(1) / scale[g];
    T(*sL)[K] = sLs;
    T(*sD)[3][KD] = sDs;
    for (int idx = hl; idx < K; idx += LPL) sL[w][idx] = Lc[g * Kp + idx] * gnorm<T>(idx);
    __syncwarp();
    {
        const T* wl = sL[w];
        auto Wc = [&](int n, int k) -> T { return (k >= 0 && k <= n) ? wl[n * n + n + k] : T(0); };  // cos-type weight (order k >= 0)
        auto Ws = [&](int n, int k) -> T { return (k >= 1 && k <= n) ? wl[n * n + n - k] : T(0); };  // sin-type weight (order -k)
        for (int idx = hl; field != nullptr && idx < P * P; idx += LPL) {  // potential only: no derived expansions
            int n1, m1;
            idx_to_nm(idx, n1, m1);
            const int n = n1 + 1, k = m1 < 0 ? -m1 : m1;
            T dx, dy, dz;
            if (m1 >= 0) {  // coefficient of R^_{n-1}^{k}
                dx = T(0.5) * Wc(n, k + 1) - (k >= 2 ? T(0.5) * Wc(n, k - 1) : (k == 1 ? Wc(n, 0) : T(0)));
                dy = -T(0.5) * Ws(n, k + 1) - (k >= 2 ? T(0.5) * Ws(n, k - 1) : T(0));
                dz = Wc(n, k);
            } else {        // coefficient of R^_{n-1}^{-k}
                dx = T(0.5) * Ws(n, k + 1) - (k >= 2 ? T(0.5) * Ws(n, k - 1) : T(0));
                dy = T(0.5) * Wc(n, k + 1) + (k >= 2 ? T(0.5) * Wc(n, k - 1) : Wc(n, 0));
                dz = Ws(n, k);
            }
            sD[w][0][idx] = dx;
            sD[w][1][idx] = dy;
            sD[w][2][idx] = dz;
        }
    }
    __syncwarp();
    for (int base = 0; base < cnt; base += LPL) {
        const int i = base + hl;
        if (i < cnt) {
            const typename V4<T>::type v = pq[st + i];
            const T x = (T)((double)v.x - cx) * inva, y = (T)((double)v.y - cy) * inva, z = (T)((double)v.z - cz) * inva;
            T phi = 0, gx = 0, gy = 0, gz = 0;
            regular_rec<P, T>(x, y, z, [&](int n, int m, T R) {
                const int idx = n * n + n + m;
                phi += sL[w][idx] * R;
                if (n < P && field != nullptr) {
                    gx += sD[w][0][idx] * R;
                    gy += sD[w][1][idx] * R;
                    gz += sD[w][2][idx] * R;
                }
            });
            // finalize (a10): add the near field written by P2P; u = -(phi_far + phi_near)/4pi (eqs. (2), (9), (14)),
            // field = -grad u = (grad phi_far + grad phi_near)/4pi (reading S2); scatter back to input order
            const typename V4<T>::type nr = near[st + i];
            const T inv4pi = T(0.079577471545947667884441881686257);
            const int64_t io = perm[st + i];
            if (pot) pot[io] = -(phi + nr.x) * inv4pi;
            if (field) {
                field[3 * io] = (gx * inva + nr.y) * inv4pi;
                field[3 * io + 1] = (gy * inva + nr.z) * inv4pi;
                field[3 * io + 2] = (gz * inva + nr.w) * inv4pi;
            }
        }
    }
}


// ------------------------------------------------------------------------------------------------ dipole sources (adjoint of the field)
// fmm_evaluate_adjoint with a field cotangent fbar: field = -grad u, so its transpose makes every target a DIPOLE source of moment
// -fbar_i: the potential it causes at x is fbar_i . grad_y (1/|x - y|) ... with the overall sign bookkeeping of evaluate():
//     phi(x) += -fbar_i . (x - y_i) / |x - y_i|^3        (near field, p2p_k<T, true>)
//     M_n^m  += -fbar_i . grad Rn_n^m((y_i - c)/a) / a   (far field, p2m_dipole_k: the transposed "L2P with gradient")
// grad R^ comes from the ladder identities of App. A.3 (the same ones l2p_k uses, pinned in tests/test_oracle_basis.py):
//     d/dz R^_n^(+-j) = R^_(n-1)^(+-j)
//     d/dx R^_n^j  = (j >= 1 ? 1/2 R^_(n-1)^(j-1) : 0) - (j >= 1 ? 1/2 : 1) R^_(n-1)^(j+1)              (j >= 0)
//     d/dx R^_n^-j = (j >= 2 ? 1/2 R^_(n-1)^-(j-1) : 0) - 1/2 R^_(n-1)^-(j+1)                            (j >= 1)
//     d/dy R^_n^j  = (j >= 2 ? 1/2 R^_(n-1)^-(j-1) : 0) + (j >= 1 ? 1/2 : 1) R^_(n-1)^-(j+1)            (j >= 0)
//     d/dy R^_n^-j = -1/2 R^_(n-1)^(j-1) - 1/2 R^_(n-1)^(j+1)                                            (j >= 1)
// with R^_(n-1)^k := 0 for |k| > n-1.
template <typename T>
__global__ void permute_dip_k(const T* __restrict__ fbar, const int32_t* __restrict__ perm, typename V4<T>::type* __restrict__ dip, int64_t N) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int64_t i = perm[k];
    dip[k] = make4<T>(fbar[3 * i], fbar[3 * i + 1], fbar[3 * i + 2], T(0));
}

template <typename T, int P>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) p2m_dipole_k(const typename V4<T>::type* __restrict__ pq, const typename V4<T>::type* __restrict__ dip,
                                                                     const int32_t* __restrict__ box_start, const int32_t* __restrict__ box_count,
                                                                     const double* __restrict__ ctr, const T* __restrict__ scale, int64_t leaf0, int64_t n_leaves,
                                                                     int Kp, T* __restrict__ Mc) {
    constexpr int KD = P > 0 ? P * P : 1;  // R^ of degree <= P-1
    const int lane = threadIdx.x & 31;
    const int64_t leaf = (int64_t)blockIdx.x * WARPS_PER_BLOCK + (threadIdx.x >> 5);
    if (leaf >= n_leaves || P == 0) return;
    const int64_t g = leaf0 + leaf;
    const int st = box_start[g], cnt = box_count[g];
    const double cx = ctr[3 * g], cy = ctr[3 * g + 1], cz = ctr[3 * g + 2];
    const T inva = T(1) / scale[g];
    for (int base = 0; base < cnt; base += 32) {
        const int i = base + lane;
        T x = 0, y = 0, z = 0, fx = 0, fy = 0, fz = 0;
        if (i < cnt) {
            const typename V4<T>::type v = pq[st + i], d = dip[st + i];
            x = (T)((double)v.x - cx) * inva; y = (T)((double)v.y - cy) * inva; z = (T)((double)v.z - cz) * inva;
            fx = d.x; fy = d.y; fz = d.z;
        }
        T R[KD];
        regular_rec<(P > 0 ? P - 1 : 0), T>(x, y, z, [&](int n, int m, T val) { R[n * n + n + m] = val; });
        auto Rl = [&](int n1, int k) -> T { return (k >= -n1 && k <= n1) ? R[n1 * n1 + n1 + k] : T(0); };
        for (int n = 1; n <= P; ++n)
            for (int m = -n; m <= n; ++m) {
                const int j = m < 0 ? -m : m, n1 = n - 1;
                T gx, gy, gz;
                if (m >= 0) {
                    gx = (j >= 1 ? T(0.5) * Rl(n1, j - 1) : T(0)) - (j >= 1 ? T(0.5) : T(1)) * Rl(n1, j + 1);
                    gy = (j >= 2 ? T(0.5) * Rl(n1, -(j - 1)) : T(0)) + (j >= 1 ? T(0.5) : T(1)) * Rl(n1, -(j + 1));
                    gz = Rl(n1, j);
                } else {
                    gx = (j >= 2 ? T(0.5) * Rl(n1, -(j - 1)) : T(0)) - T(0.5) * Rl(n1, -(j + 1));
                    gy = -T(0.5) * Rl(n1, j - 1) - T(0.5) * Rl(n1, j + 1);
                    gz = Rl(n1, -j);
                }
                T v = -(fx * gx + fy * gy + fz * gz);
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
                const int idx = n * n + n + m;
                if (lane == 0) Mc[g * Kp + idx] += v * inva * gnorm<T>(idx);
            }
    }
}

// ------------------------------------------------------------------------------------------------ generic translations
// One warp per translation; state vectors in shared memory; rotation = Z(-phi) B Z(-theta) B^T [shift] B Z(theta) B^T Z(phi).
template <typename T>
struct WarpScratch {
    T v[KMAX], u[KMAX];
    T cph[PMAX + 1], sph[PMAX + 1], cth[PMAX + 1], sth[PMAX + 1], pw1[PMAX + 1], pw2[PMAX + 1];
};

struct TabPtrs {
    const void* B;  // T-typed rotation blocks
    const double *H, *A;
};

template <typename T>
__device__ inline void az_step(int K, const T* in, T* out, const T* c, const T* s, T sign, int lane) {
    for (int idx = lane; idx < K; idx += 32) {
        int n, m;
        idx_to_nm(idx, n, m);
        const int am = m < 0 ? -m : m;
        T ss = sign * s[am];
        if (m < 0) ss = -ss;
        out[idx] = in[idx] * c[am] - in[idx - 2 * m] * ss;
    }
}

template <typename T>
__device__ inline void b_step(int K, const T* in, T* out, const T* Btab, bool transpose, int lane) {
    for (int idx = lane; idx < K; idx += 32) {
        int n, m;
        idx_to_nm(idx, n, m);
        const int w = 2 * n + 1, i = m + n;
        const T* Bn = Btab + boff(n);
        const T* vin = in + n * n;
        T acc = 0;
        if (transpose) for (int j = 0; j < w; ++j) acc += Bn[j * w + i] * vin[j];
        else for (int j = 0; j < w; ++j) acc += Bn[i * w + j] * vin[j];
        out[idx] = acc;
    }
}

// kind 0 = M2M (b = child - parent), 1 = M2L (b = source - target), 2 = L2L (b = parent - child)   [reading G3]
// a_old / a_new: length scales of the box the input / the output expansion belongs to.  Result in ws.u.
template <typename T>
__device__ inline void translate_warp(int kind, int p, const T* __restrict__ src, double bxd, double byd, double bzd, T a_old, T a_new,
                                      WarpScratch<T>& ws, TabPtrs tp, int lane) {
    const int K = (p + 1) * (p + 1);
    const int P1 = PMAX + 1;
    const T bx = (T)bxd, by = (T)byd, bz = (T)bzd;
    const T r = sqrt(bx * bx + by * by + bz * bz);
    const T rxy = sqrt(bx * bx + by * by);
    const T ct = r > 0 ? bz / r : T(1), st = r > 0 ? rxy / r : T(0);
    const T cp = rxy > 0 ? bx / rxy : T(1), sp = rxy > 0 ? by / rxy : T(0);
    for (int idx = lane; idx < K; idx += 32) ws.v[idx] = src[idx];
    if (lane <= p) {
        T c = 1, s = 0, c2 = 1, s2 = 0, x1, x2, p1 = 1, p2 = 1;
        if (kind == 0) { x1 = r / a_new; x2 = a_old / a_new; }
        else if (kind == 1) { x1 = a_new / r; x2 = a_old / r; }
        else { x1 = -r / a_old; x2 = a_new / a_old; }
        for (int i = 0; i < lane; ++i) {
            T t = c * cp - s * sp; s = s * cp + c * sp; c = t;
            t = c2 * ct - s2 * st; s2 = s2 * ct + c2 * st; c2 = t;
            p1 *= x1; p2 *= x2;
        }
        ws.cph[lane] = c; ws.sph[lane] = s; ws.cth[lane] = c2; ws.sth[lane] = s2; ws.pw1[lane] = p1; ws.pw2[lane] = p2;
    }
    __syncwarp();
    const T* Btab = (const T*)tp.B;
    az_step<T>(K, ws.v, ws.u, ws.cph, ws.sph, T(1), lane); __syncwarp();
    b_step<T>(K, ws.u, ws.v, Btab, true, lane); __syncwarp();
    az_step<T>(K, ws.v, ws.u, ws.cth, ws.sth, T(1), lane); __syncwarp();
    b_step<T>(K, ws.u, ws.v, Btab, false, lane); __syncwarp();
    // z-shift (App. B.3) in the normalised, scaled representation
    for (int idx = lane; idx < K; idx += 32) {
        int n, m;
        idx_to_nm(idx, n, m);
        const int am = m < 0 ? -m : m;
        T acc = 0;
        if (kind == 0) {
            for (int k = am; k <= n; ++k) acc += (T)tp.A[(am * P1 + n) * P1 + k] * ws.pw1[n - k] * ws.pw2[k] * ws.v[k * k + k + m];
        } else if (kind == 1) {
            for (int k = am; k <= p; ++k) acc += (T)tp.H[(am * P1 + n) * P1 + k] * ws.pw2[k] * ws.v[k * k + k + m];
            acc *= ws.pw1[n] / r;
        } else {
            for (int k = n; k <= p; ++k) acc += (T)tp.A[(am * P1 + k) * P1 + n] * ws.pw1[k - n] * ws.v[k * k + k + m];
            acc *= ws.pw2[n];
        }
        ws.u[idx] = acc;
    }
    __syncwarp();
    b_step<T>(K, ws.u, ws.v, Btab, true, lane); __syncwarp();
    az_step<T>(K, ws.v, ws.u, ws.cth, ws.sth, T(-1), lane); __syncwarp();
    b_step<T>(K, ws.u, ws.v, Btab, false, lane); __syncwarp();
    az_step<T>(K, ws.v, ws.u, ws.cph, ws.sph, T(-1), lane); __syncwarp();
}

constexpr int NJMAX = (KMAX + 31) / 32;

// M2M (a5): warp per parent box of level l-1, children in ascending order
template <typename T>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) m2m_k(int p, int s, int64_t off_parent, int64_t off_child, int64_t nb_parent,
                                                              const int32_t* __restrict__ box_count, const double* __restrict__ ctr,
                                                              const T* __restrict__ scale, int Kp, T* __restrict__ Mc, TabPtrs tp) {
    __shared__ WarpScratch<T> wsm[WARPS_PER_BLOCK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t bp = (int64_t)blockIdx.x * WARPS_PER_BLOCK + w;
    if (bp >= nb_parent) return;
    const int K = (p + 1) * (p + 1);
    const int64_t gp = off_parent + bp;
    T acc[NJMAX];
#pragma unroll
    for (int j = 0; j < NJMAX; ++j) acc[j] = 0;
    for (int j = 0; j < (1 << s); ++j) {
        const int64_t gc = off_child + (bp << s) + j;
        if (box_count[gc] == 0) continue;
        translate_warp<T>(0, p, Mc + gc * Kp, ctr[3 * gc] - ctr[3 * gp], ctr[3 * gc + 1] - ctr[3 * gp + 1], ctr[3 * gc + 2] - ctr[3 * gp + 2],
                          scale[gc], scale[gp], wsm[w], tp, lane);
#pragma unroll
        for (int jj = 0; jj < NJMAX; ++jj) {
            const int idx = lane + 32 * jj;
            if (idx < K) acc[jj] += wsm[w].u[idx];
        }
        __syncwarp();
    }
#pragma unroll
    for (int jj = 0; jj < NJMAX; ++jj) {
        const int idx = lane + 32 * jj;
        if (idx < K) Mc[gp * Kp + idx] = acc[jj];
    }
}

// M2L (a6), generic: warp per target box, loop over its row of the weak list (CSR by target)
template <typename T>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) m2l_generic_k(int p, int64_t n_boxes, const int64_t* __restrict__ weak_off,
                                                                      const int32_t* __restrict__ weak_src, const double* __restrict__ ctr,
                                                                      const T* __restrict__ scale, const double* __restrict__ ctr_s,
                                                                      const T* __restrict__ scale_s, int Kp, const T* __restrict__ Mc,
                                                                      T* __restrict__ Lc, TabPtrs tp) {
    __shared__ WarpScratch<T> wsm[WARPS_PER_BLOCK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t gt = (int64_t)blockIdx.x * WARPS_PER_BLOCK + w;
    if (gt >= n_boxes) return;
    const int64_t e0 = weak_off[gt], e1 = weak_off[gt + 1];
    if (e0 == e1) return;
    const int K = (p + 1) * (p + 1);
    T acc[NJMAX];
#pragma unroll
    for (int j = 0; j < NJMAX; ++j) acc[j] = 0;
    const double tx = ctr[3 * gt], ty = ctr[3 * gt + 1], tz = ctr[3 * gt + 2];
    const T at = scale[gt];
    for (int64_t e = e0; e < e1; ++e) {
        const int64_t gs = weak_src[e];
        translate_warp<T>(1, p, Mc + gs * Kp, ctr_s[3 * gs] - tx, ctr_s[3 * gs + 1] - ty, ctr_s[3 * gs + 2] - tz, scale_s[gs], at, wsm[w], tp, lane);
#pragma unroll
        for (int jj = 0; jj < NJMAX; ++jj) {
            const int idx = lane + 32 * jj;
            if (idx < K) acc[jj] += wsm[w].u[idx];
        }
        __syncwarp();
    }
#pragma unroll
    for (int jj = 0; jj < NJMAX; ++jj) {
        const int idx = lane + 32 * jj;
        if (idx < K) Lc[gt * Kp + idx] += acc[jj];
    }
}

// L2L (a7): warp per child box of level l
template <typename T>
__global__ void __launch_bounds__(WARPS_PER_BLOCK * 32) l2l_k(int p, int s, int64_t off_parent, int64_t off_child, int64_t nb_child,
                                                              const int32_t* __restrict__ box_count, const double* __restrict__ ctr,
                                                              const T* __restrict__ scale, int Kp, T* __restrict__ Lc, TabPtrs tp) {
    __shared__ WarpScratch<T> wsm[WARPS_PER_BLOCK];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t bc = (int64_t)blockIdx.x * WARPS_PER_BLOCK + w;
    if (bc >= nb_child) return;
    const int64_t gc = off_child + bc, gp = off_parent + (bc >> s);
    if (box_count[gc] == 0) return;
    const int K = (p + 1) * (p + 1);
    translate_warp<T>(2, p, Lc + gp * Kp, ctr[3 * gp] - ctr[3 * gc], ctr[3 * gp + 1] - ctr[3 * gc + 1], ctr[3 * gp + 2] - ctr[3 * gc + 2],
                      scale[gp], scale[gc], wsm[w], tp, lane);
    for (int idx = lane; idx < K; idx += 32) Lc[gc * Kp + idx] += wsm[w].u[idx];
}

// ------------------------------------------------------------------------------------------------ P2P (a9)
// One target leaf per CTA.  Threads are arranged as (target group, source slice): each thread keeps TPT targets in
// registers and walks every nslices-th source of the shared-memory tile; partial sums are combined through shared memory.
constexpr int P2P_THREADS = 128;
constexpr int P2P_TPT = 4;
constexpr int P2P_TILE = 512;

// DIP: every source also carries a dipole (dip_s, see above); potential only
template <typename T, bool DIP>
__global__ void __launch_bounds__(P2P_THREADS) p2p_k(const typename V4<T>::type* __restrict__ pq, const int32_t* __restrict__ leaf_start,
                                                     const int32_t* __restrict__ leaf_cnt, const typename V4<T>::type* __restrict__ pq_s,
                                                     const int32_t* __restrict__ sleaf_start, const int32_t* __restrict__ sleaf_cnt,
                                                     const int64_t* __restrict__ strong_off, const int32_t* __restrict__ strong_src,
                                                     typename V4<T>::type* __restrict__ near,  // *_s: the sources' hierarchy (== the targets' unless PAPER.md:82)
                                                     const typename V4<T>::type* __restrict__ dip_s) {
    using T4 = typename V4<T>::type;
    __shared__ T4 sh[P2P_TILE];
    __shared__ T4 shd[DIP ? P2P_TILE : 1];
    __shared__ T red[P2P_THREADS * P2P_TPT * 4];
    const int tid = threadIdx.x;
    const int64_t leaf = blockIdx.x;
    const int tst = leaf_start[leaf], tcnt = leaf_cnt[leaf];
    if (tcnt == 0) return;
    const int64_t e0 = strong_off[leaf], e1 = strong_off[leaf + 1];
    for (int tbase = 0; tbase < tcnt; tbase += P2P_THREADS * P2P_TPT) {
        const int tn = min(tcnt - tbase, P2P_THREADS * P2P_TPT);
        int ntg = (tn + P2P_TPT - 1) / P2P_TPT, ntgp = 1;
        while (ntgp < ntg) ntgp <<= 1;
        const int nsl = P2P_THREADS / ntgp;
        const int tg = tid & (ntgp - 1), sl = tid / ntgp;
        T tx[P2P_TPT], ty[P2P_TPT], tz[P2P_TPT], ph[P2P_TPT], gx[P2P_TPT], gy[P2P_TPT], gz[P2P_TPT];
#pragma unroll
        for (int t = 0; t < P2P_TPT; ++t) {
            const int ti = tg * P2P_TPT + t;
            // out-of-range targets are parked far away with zero weight (their sums are discarded)
            if (ti < tn) {
                const T4 v = pq[tst + tbase + ti];
                tx[t] = v.x; ty[t] = v.y; tz[t] = v.z;
            } else {
                tx[t] = T(1e18); ty[t] = T(1e18); tz[t] = T(1e18);
            }
            ph[t] = gx[t] = gy[t] = gz[t] = T(0);
        }
        int64_t e = e0;
        int sub = 0;
        for (;;) {
            int tile_n = 0;
            __syncthreads();
            while (e < e1 && tile_n < P2P_TILE) {
                const int sleaf = strong_src[e];
                const int sst = sleaf_start[sleaf], sc = sleaf_cnt[sleaf];
                const int take = min(sc - sub, P2P_TILE - tile_n);
                for (int i = tid; i < take; i += P2P_THREADS) {
                    sh[tile_n + i] = pq_s[sst + sub + i];
                    if constexpr (DIP) shd[tile_n + i] = dip_s[sst + sub + i];
                }
                tile_n += take;
                sub += take;
                if (sub >= sc) { ++e; sub = 0; }
            }
            if (tile_n == 0) break;
            __syncthreads();
#pragma unroll 2
            for (int j = sl; j < tile_n; j += nsl) {
                const T4 sv = sh[j];
#pragma unroll
                for (int t = 0; t < P2P_TPT; ++t) {
                    const T dx = tx[t] - sv.x, dy = ty[t] - sv.y, dz = tz[t] - sv.z;
                    const T r2 = fma(dz, dz, fma(dy, dy, dx * dx));  // the same order as the packed kernel (p2p_fast.cu)
                    T inv = rsqrt_t<T>(r2);
                    // S3: self / coincident pairs contribute nothing; in fp32 every pair with r^2 below the smallest normal number
                    // counts as coincident (its 1/r^3 is not representable), in fp64 only r^2 == 0
                    inv = (r2 >= r2_min<T>()) ? inv : T(0);
                    const T inv2 = inv * inv;
                    const T q3 = sv.w * inv * inv2;
                    ph[t] += sv.w * inv;
                    if constexpr (DIP) {
                        const T4 dv = shd[j];
                        ph[t] -= (dv.x * dx + dv.y * dy + dv.z * dz) * (inv * inv2);
                    } else {
                        gx[t] -= q3 * dx; gy[t] -= q3 * dy; gz[t] -= q3 * dz;
                    }
                }
            }
        }
        // combine the source slices
        __syncthreads();
#pragma unroll
        for (int t = 0; t < P2P_TPT; ++t) {
            T* r = red + ((sl * ntgp + tg) * P2P_TPT + t) * 4;
            r[0] = ph[t]; r[1] = gx[t]; r[2] = gy[t]; r[3] = gz[t];
        }
        __syncthreads();
        for (int ti = tid; ti < tn; ti += P2P_THREADS) {
            const int g2 = ti / P2P_TPT, t2 = ti % P2P_TPT;
            T a0 = 0, a1 = 0, a2 = 0, a3 = 0;
            for (int s2 = 0; s2 < nsl; ++s2) {
                const T* r = red + ((s2 * ntgp + g2) * P2P_TPT + t2) * 4;
                a0 += r[0]; a1 += r[1]; a2 += r[2]; a3 += r[3];
            }
            near[tst + tbase + ti] = make4<T>(a0, a1, a2, a3);  // (phi_near, grad phi_near), tree order
        }
    }
}

// leaves [lo, hi) of the leaf level (hi < 0: all)
template <typename T, int P, int LPL>
void launch_p2m_l2p_t(const Plan& Pl, bool l2p, void* d_pot, void* d_field, cudaStream_t st, int64_t lo, int64_t hi) {
    using T4 = typename V4<T>::type;
    if (hi < 0) { lo = 0; hi = Pl.n_leaves; }
    if (hi <= lo) return;
    const int64_t leaf0 = Pl.level_off[Pl.L] + lo, nl = hi - lo;
    const unsigned grid = nblocks(nl, WARPS_PER_BLOCK * (32 / LPL));
    if (!l2p)
        p2m_k<T, P, LPL><<<grid, WARPS_PER_BLOCK * 32, 0, st>>>((const T4*)Pl.pq.p, Pl.box_start.p, Pl.box_count.p, Pl.box_ctr.p,
                                                                (const T*)Pl.box_scale.p, leaf0, nl, Pl.Kp, (T*)Pl.Mc.p);
    else
        l2p_k<T, P, LPL><<<grid, WARPS_PER_BLOCK * 32, 0, st>>>((const T4*)Pl.pq.p, Pl.box_start.p, Pl.box_count.p, Pl.box_ctr.p,
                                                                (const T*)Pl.box_scale.p, leaf0, nl, Pl.Kp, (const T*)Pl.Lc.p,
                                                                (const T4*)Pl.near.p, Pl.perm.p, (T*)d_pot, (T*)d_field);
}

template <typename T, int P>
void launch_p2m_l2p(const Plan& Pl, bool l2p, void* d_pot, void* d_field, cudaStream_t st, int64_t lo, int64_t hi) {
    // leaves of <= 16 particles (e.g. config 4: N_max = 64, s = 3): two leaves per warp.  fp32, p <= 8 only (compile time).
    if constexpr (sizeof(T) == 4 && P <= 8) {
        if (Pl.max_leaf <= 16) { launch_p2m_l2p_t<T, P, 16>(Pl, l2p, d_pot, d_field, st, lo, hi); return; }
    }
    launch_p2m_l2p_t<T, P, 32>(Pl, l2p, d_pot, d_field, st, lo, hi);
}

template <typename T>
void dispatch_p2m_dipole(const Plan& Pl, cudaStream_t st) {
    using T4 = typename V4<T>::type;
    const unsigned grid = nblocks(Pl.n_leaves, WARPS_PER_BLOCK);
    switch (Pl.p) {
#define FMM_CASE(PP) case PP: p2m_dipole_k<T, PP><<<grid, WARPS_PER_BLOCK * 32, 0, st>>>((const T4*)Pl.pq.p, (const T4*)Pl.dip.p, Pl.box_start.p, Pl.box_count.p, \
            Pl.box_ctr.p, (const T*)Pl.box_scale.p, Pl.level_off[Pl.L], Pl.n_leaves, Pl.Kp, (T*)Pl.Mc.p); break;
        FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
        FMM_CASE(9) FMM_CASE(10) FMM_CASE(11) FMM_CASE(12) FMM_CASE(13) FMM_CASE(14) FMM_CASE(15) FMM_CASE(16)
#undef FMM_CASE
        default: break;  // p = 0: a dipole has no monopole moment
    }
}

template <typename T>
void dispatch_p2m_l2p(const Plan& Pl, bool l2p, void* d_pot, void* d_field, cudaStream_t st, int64_t lo = 0, int64_t hi = -1) {
    switch (Pl.p) {
#define FMM_CASE(PP) case PP: launch_p2m_l2p<T, PP>(Pl, l2p, d_pot, d_field, st, lo, hi); break;
        FMM_CASE(0) FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
        FMM_CASE(9) FMM_CASE(10) FMM_CASE(11) FMM_CASE(12) FMM_CASE(13) FMM_CASE(14) FMM_CASE(15) FMM_CASE(16)
#undef FMM_CASE
    }
}

// __constant__ copies of g_n^m: one upload per device
void ensure_constants(const Plan& P) {
    DeviceCtx& ctx = device_ctx(P.device);
    std::lock_guard<std::mutex> lock(ctx.mu);
    if (!ctx.const_uploaded) {
        std::vector<double> g(KMAX);
        std::vector<float> gf(KMAX);
        FMM_CUDA_CHECK(cudaMemcpy(g.data(), ctx.tab.d_g, KMAX * sizeof(double), cudaMemcpyDeviceToHost));
        for (int i = 0; i < KMAX; ++i) gf[i] = (float)g[i];
        FMM_CUDA_CHECK(cudaMemcpyToSymbol(c_g, g.data(), KMAX * sizeof(double)));
        FMM_CUDA_CHECK(cudaMemcpyToSymbol(c_gf, gf.data(), KMAX * sizeof(float)));
        ctx.const_uploaded = true;
    }
}

// Internal streams of a plan (created on first use).  s_far / s_up have the highest priority, s_near the lowest, so that
// the latency-bound far-field kernels get SM resources as soon as they are launched and P2P fills whatever is left.
void ensure_streams(const Plan& Pl) {
    if (Pl.s_far) return;
    int lo = 0, hi = 0;
    FMM_CUDA_CHECK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    FMM_CUDA_CHECK(cudaStreamCreateWithPriority(&Pl.s_far, cudaStreamNonBlocking, hi));
    FMM_CUDA_CHECK(cudaStreamCreateWithPriority(&Pl.s_up, cudaStreamNonBlocking, hi));
    FMM_CUDA_CHECK(cudaStreamCreateWithPriority(&Pl.s_near, cudaStreamNonBlocking, lo));
    for (cudaEvent_t* e : {&Pl.e_fork, &Pl.e_perm, &Pl.e_p2m, &Pl.e_up, &Pl.e_near, &Pl.e_done})
        FMM_CUDA_CHECK(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
}

// Separate sources and targets (fmm_plan_create_targets): Pl holds the targets' hierarchy, Pl.S the sources'.
// permute + P2M + M2M run on the source hierarchy, the M2L joins the two, L2L + L2P run on the target hierarchy and the P2P sums
// source leaves into target leaves.  Weak pairs may join any two levels, so the whole upward pass precedes the M2L; the P2P
// still runs beside the far-field chain on its own stream.  ev != nullptr: serial, one event per stage (same order as run_t).
template <typename T>
void run_st(const Plan& Pl, const void* d_q, void* d_pot, void* d_field, cudaStream_t st, cudaEvent_t* ev, const void* d_dip) {
    using T4 = typename V4<T>::type;
    const Plan& S = *Pl.S;
    const Tables& tb = tables(Pl.device);
    TabPtrs tp{sizeof(T) == 4 ? (const void*)tb.d_Bf : (const void*)tb.d_B, tb.d_H, tb.d_A};
    const int p = Pl.p, s = Pl.s;
    const bool serial = ev != nullptr || Pl.serial || Pl.deterministic;
    cudaStream_t sF = st, sN = st;
    if (!serial) {
        ensure_streams(Pl);
        sF = Pl.s_far; sN = Pl.s_near;
        FMM_CUDA_CHECK(cudaEventRecord(Pl.e_fork, st));
        FMM_CUDA_CHECK(cudaStreamWaitEvent(sF, Pl.e_fork, 0));
    }
    auto mark = [&](int i) { if (ev) FMM_CUDA_CHECK(cudaEventRecord(ev[i], st)); };
    auto after = [&](cudaStream_t waiter, cudaStream_t producer, cudaEvent_t e) {
        if (serial) return;
        FMM_CUDA_CHECK(cudaEventRecord(e, producer));
        FMM_CUDA_CHECK(cudaStreamWaitEvent(waiter, e, 0));
    };
    const bool fast = Pl.m2l_variant != 1 && xlate_fast_available(p, Pl.dtype);
    const bool fast_p2p = sizeof(T) == 4 && Pl.m2l_variant != 1;
    const int64_t leaf0 = Pl.level_off[Pl.L], sleaf0 = S.level_off[S.L];
    auto launch_p2p = [&](cudaStream_t q) {
        if (d_dip)
            p2p_k<T, true><<<(unsigned)Pl.n_leaves, P2P_THREADS, 0, q>>>((const T4*)Pl.pq.p, Pl.box_start.p + leaf0, Pl.box_count.p + leaf0, (const T4*)S.pq.p,
                                                                        S.box_start.p + sleaf0, S.box_count.p + sleaf0, Pl.strong_off.p, Pl.strong_src.p,
                                                                        (T4*)Pl.near.p, (const T4*)S.dip.p);
        else if (fast_p2p) p2p_fast_launch(Pl, q, d_field != nullptr);
        else if (sizeof(T) == 8 && Pl.m2l_variant != 1) p2p_fast64_launch(Pl, q, d_field != nullptr);
        else p2p_k<T, false><<<(unsigned)Pl.n_leaves, P2P_THREADS, 0, q>>>((const T4*)Pl.pq.p, Pl.box_start.p + leaf0, Pl.box_count.p + leaf0, (const T4*)S.pq.p,
                                                                         S.box_start.p + sleaf0, S.box_count.p + sleaf0, Pl.strong_off.p, Pl.strong_src.p,
                                                                         (T4*)Pl.near.p, nullptr);
        FMM_CUDA_CHECK(cudaGetLastError());
    };
    mark(0);
    permute_k<T><<<nblocks(S.N, 256), 256, 0, sF>>>((const T*)S.pos_tree.p, (const T*)d_q, S.perm.p, (T4*)S.pq.p, S.src_slot.p,
                                                    sizeof(T) == 4 ? S.srcg.p : nullptr, S.N);
    FMM_CUDA_CHECK(cudaGetLastError());
    permute_k<T><<<nblocks(Pl.N, 256), 256, 0, sF>>>((const T*)Pl.pos_tree.p, nullptr, Pl.perm.p, (T4*)Pl.pq.p, nullptr, nullptr, Pl.N);
    FMM_CUDA_CHECK(cudaGetLastError());
    if (d_dip) {
        if (!S.dip.p) S.dip.alloc((size_t)S.N * 4 * sizeof(T));
        permute_dip_k<T><<<nblocks(S.N, 256), 256, 0, sF>>>((const T*)d_dip, S.perm.p, (T4*)S.dip.p, S.N);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    after(sN, sF, Pl.e_perm);
    if (!serial) launch_p2p(sN);
    FMM_CUDA_CHECK(cudaMemsetAsync(Pl.Lc.p, 0, Pl.Lc.n, sF));
    mark(1);
    dispatch_p2m_l2p<T>(S, false, nullptr, nullptr, sF);
    if (d_dip) dispatch_p2m_dipole<T>(S, sF);
    FMM_CUDA_CHECK(cudaGetLastError());
    mark(2);
    if (fast && S.L > 0) FMM_CUDA_CHECK(cudaMemsetAsync(S.Mc.p, 0, (size_t)S.level_off[S.L] * S.Kp * sizeof(T), sF));
    for (int l = S.L; l >= 1; --l) {
        if (fast) { xlate_fast_launch(S, 0, l, sF); continue; }
        const int64_t nbp = (int64_t)1 << (s * (l - 1));
        m2m_k<T><<<nblocks(nbp, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, sF>>>(p, s, S.level_off[l - 1], S.level_off[l], nbp, S.box_count.p, S.box_ctr.p,
                                                                                (const T*)S.box_scale.p, S.Kp, (T*)S.Mc.p, tp);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    mark(3);
    if (Pl.n_weak > 0) {
        // deterministic: one warp per target row (p <= 8) or the generic warp-per-box kernel -- both sum a row in list order
        if (fast && Pl.deterministic && m2l_row_available(p, Pl.dtype)) m2l_row_launch(Pl, sF);
        else if (fast && !Pl.deterministic) xlate_fast_launch(Pl, 1, 0, sF, 0, Pl.n_weak);
        else
            m2l_generic_k<T><<<nblocks(Pl.n_boxes, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, sF>>>(
                p, Pl.n_boxes, Pl.weak_off.p, Pl.weak_src.p, Pl.box_ctr.p, (const T*)Pl.box_scale.p, S.box_ctr.p, (const T*)S.box_scale.p, Pl.Kp,
                (const T*)S.Mc.p, (T*)Pl.Lc.p, tp);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    mark(4);
    for (int l = 1; l <= Pl.L; ++l) {
        if (fast) { xlate_fast_launch(Pl, 2, l, sF); continue; }
        const int64_t nbc = (int64_t)1 << (s * l);
        l2l_k<T><<<nblocks(nbc, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, sF>>>(p, s, Pl.level_off[l - 1], Pl.level_off[l], nbc, Pl.box_count.p, Pl.box_ctr.p,
                                                                                (const T*)Pl.box_scale.p, Pl.Kp, (T*)Pl.Lc.p, tp);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    mark(5);
    if (serial) launch_p2p(st);
    else after(sF, sN, Pl.e_near);
    mark(6);
    dispatch_p2m_l2p<T>(Pl, true, d_pot, d_field, sF);
    FMM_CUDA_CHECK(cudaGetLastError());
    mark(7);
    after(st, sF, Pl.e_done);
}

// One evaluate.  ev == nullptr: the production schedule -- three internal streams forked from / joined to the caller's
// stream: far chain (permute, P2M, leaf-level M2L, L2P + finalize), tree chain (M2M levels, the M2L of the upper levels, then
// the L2L levels, all concurrent with the leaf-level M2L) and near field (P2P, concurrent with everything between permute and L2P).
// ev != nullptr: the same kernels back to back on the caller's stream with an event after every stage (profiling).
template <typename T>
void run_t(const Plan& Pl, const void* d_q, void* d_pot, void* d_field, cudaStream_t st, cudaEvent_t* ev, const void* d_dip) {
    using T4 = typename V4<T>::type;
    const Tables& tb = tables(Pl.device);
    TabPtrs tp{sizeof(T) == 4 ? (const void*)tb.d_Bf : (const void*)tb.d_B, tb.d_H, tb.d_A};
    const int p = Pl.p, s = Pl.s, L = Pl.L;
    const int64_t N = Pl.N;
    const bool serial = ev != nullptr || Pl.serial || Pl.deterministic;
    cudaStream_t sF = st, sU = st, sN = st;
    if (!serial) {
        ensure_streams(Pl);
        sF = Pl.s_far; sU = Pl.s_up; sN = Pl.s_near;
        FMM_CUDA_CHECK(cudaEventRecord(Pl.e_fork, st));
        FMM_CUDA_CHECK(cudaStreamWaitEvent(sF, Pl.e_fork, 0));
    }
    auto mark = [&](int i) { if (ev) FMM_CUDA_CHECK(cudaEventRecord(ev[i], st)); };
    auto after = [&](cudaStream_t waiter, cudaStream_t producer, cudaEvent_t e) {  // waiter continues after what producer has queued
        if (serial) return;
        FMM_CUDA_CHECK(cudaEventRecord(e, producer));
        FMM_CUDA_CHECK(cudaStreamWaitEvent(waiter, e, 0));
    };
    // m2l_variant: 0 = register / shared-memory kernels (one translation per thread), 1 = generic kernels (warp per box)
    const bool fast = Pl.m2l_variant != 1 && xlate_fast_available(p, Pl.dtype);
    const bool fast_p2p = sizeof(T) == 4 && Pl.m2l_variant != 1;
    const int64_t leaf0 = Pl.level_off[L];
    auto launch_p2p = [&](cudaStream_t q) {
        if (d_dip)
            p2p_k<T, true><<<(unsigned)Pl.n_leaves, P2P_THREADS, 0, q>>>((const T4*)Pl.pq.p, Pl.box_start.p + leaf0, Pl.box_count.p + leaf0, (const T4*)Pl.pq.p,
                                                                        Pl.box_start.p + leaf0, Pl.box_count.p + leaf0, Pl.strong_off.p, Pl.strong_src.p,
                                                                        (T4*)Pl.near.p, (const T4*)Pl.dip.p);
        else if (fast_p2p) p2p_fast_launch(Pl, q, d_field != nullptr);
        else if (sizeof(T) == 8 && Pl.m2l_variant != 1) p2p_fast64_launch(Pl, q, d_field != nullptr);
        else p2p_k<T, false><<<(unsigned)Pl.n_leaves, P2P_THREADS, 0, q>>>((const T4*)Pl.pq.p, Pl.box_start.p + leaf0, Pl.box_count.p + leaf0, (const T4*)Pl.pq.p,
                                                                         Pl.box_start.p + leaf0, Pl.box_count.p + leaf0, Pl.strong_off.p, Pl.strong_src.p,
                                                                         (T4*)Pl.near.p, nullptr);
        FMM_CUDA_CHECK(cudaGetLastError());
    };

    mark(0);
    permute_k<T><<<nblocks(N, 256), 256, 0, sF>>>((const T*)Pl.pos_tree.p, (const T*)d_q, Pl.perm.p, (T4*)Pl.pq.p, Pl.src_slot.p,
                                                  sizeof(T) == 4 ? Pl.srcg.p : nullptr, N);
    FMM_CUDA_CHECK(cudaGetLastError());
    if (d_dip) {
        if (!Pl.dip.p) Pl.dip.alloc((size_t)N * 4 * sizeof(T));
        permute_dip_k<T><<<nblocks(N, 256), 256, 0, sF>>>((const T*)d_dip, Pl.perm.p, (T4*)Pl.dip.p, N);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    after(sN, sF, Pl.e_perm);
    if (!serial) launch_p2p(sN);
    FMM_CUDA_CHECK(cudaMemsetAsync(Pl.Lc.p, 0, Pl.Lc.n, sF));
    mark(1);
    dispatch_p2m_l2p<T>(Pl, false, nullptr, nullptr, sF);
    if (d_dip) dispatch_p2m_dipole<T>(Pl, sF);
    FMM_CUDA_CHECK(cudaGetLastError());
    mark(2);
    if (fast && L > 0)  // the register kernels accumulate into the parents
        FMM_CUDA_CHECK(cudaMemsetAsync(Pl.Mc.p, 0, (size_t)Pl.level_off[L] * Pl.Kp * sizeof(T), sF));
    // the M2L of the leaf level needs only the P2M output: with the register kernels it runs on sF while M2M and the upper
    // levels' M2L run on sU (weak pairs are sorted by target id, hence by level; rows of different levels are disjoint)
    const int64_t w_leaf = (int64_t)Pl.weak_level_off.size() > L ? Pl.weak_level_off[L] : 0;
    const bool split = !serial && fast && L > 0 && !Pl.no_split;
    if (split) after(sU, sF, Pl.e_p2m);
    cudaStream_t sM = split ? sU : sF;
    for (int l = L; l > Pl.top_level; --l) {
        if (fast) { xlate_fast_launch(Pl, 0, l, sM); continue; }
        const int64_t nbp = (int64_t)1 << (s * (l - 1));
        m2m_k<T><<<nblocks(nbp, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, sM>>>(p, s, Pl.level_off[l - 1], Pl.level_off[l], nbp, Pl.box_count.p,
                                                                                Pl.box_ctr.p, (const T*)Pl.box_scale.p, Pl.Kp, (T*)Pl.Mc.p, tp);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    mark(3);
    if (Pl.n_weak > 0) {
        auto m2l_range = [&](int64_t e0, int64_t e1, cudaStream_t q) {
            if (e1 <= e0) return;
            xlate_fast_launch(Pl, 1, 0, q, e0, e1);
        };
        if (split) {
            m2l_range(w_leaf, Pl.n_weak, sF);
            m2l_range(0, w_leaf, sU);
        } else if (fast && Pl.deterministic && m2l_row_available(p, Pl.dtype)) {
            m2l_row_launch(Pl, sF);  // one warp per target row, sums in list order (see run_st)
        } else if (fast && !Pl.deterministic) {
            m2l_range(0, Pl.n_weak, sF);
        } else {
            m2l_generic_k<T><<<nblocks(Pl.n_boxes, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, sF>>>(
                p, Pl.n_boxes, Pl.weak_off.p, Pl.weak_src.p, Pl.box_ctr.p, (const T*)Pl.box_scale.p, Pl.box_ctr.p, (const T*)Pl.box_scale.p, Pl.Kp,
                (const T*)Pl.Mc.p, (T*)Pl.Lc.p, tp);
        }
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    mark(4);
    // L2L (a7).  The register kernels ADD into the children with atomics, exactly like the M2L, so in the split schedule the
    // whole downward pass runs on sU right behind the upper levels' M2L and beside the leaf-level M2L on sF.
    cudaStream_t sL = split ? sU : sF;
    for (int l = Pl.top_level + 1; l <= L; ++l) {
        if (fast) { xlate_fast_launch(Pl, 2, l, sL); continue; }
        const int64_t nbc = (int64_t)1 << (s * l);
        l2l_k<T><<<nblocks(nbc, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, sL>>>(p, s, Pl.level_off[l - 1], Pl.level_off[l], nbc, Pl.box_count.p,
                                                                                Pl.box_ctr.p, (const T*)Pl.box_scale.p, Pl.Kp, (T*)Pl.Lc.p, tp);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    if (split) after(sF, sU, Pl.e_up);
    mark(5);
    if (serial) launch_p2p(st);
    else after(sF, sN, Pl.e_near);
    mark(6);
    dispatch_p2m_l2p<T>(Pl, true, d_pot, d_field, sF);
    FMM_CUDA_CHECK(cudaGetLastError());
    mark(7);
    after(st, sF, Pl.e_done);
}


// ------------------------------------------------------------------------------------------------ target-sharded evaluate
// SURVEY 8(e) / PAPER.md:226 ("distribution of data across multiple GPUs is not yet supported"): targets are independent once the
// multipoles are known, and a contiguous range of leaves is a set of subtrees (Z-order layout).  Shard r of n owns the
// leaves [n_leaves r / n, n_leaves (r+1) / n):
//   upward   : permute all charges (they are replicated), P2M for ITS leaves only;
//   exchange : the caller all-gathers the leaf rows of the multipole array (the one data-path collective; fmm.py uses NCCL);
//   downward : M2M for all boxes (cheap, redundant), then M2L / L2L for its boxes and their ancestors only, P2P and L2P for its
//              leaves -- outputs are written for the shard's particles only.
template <typename T>
void shard_upward_t(const Plan& Pl, int64_t lo, int64_t hi, const void* d_q, cudaStream_t st) {
    using T4 = typename V4<T>::type;
    permute_k<T><<<nblocks(Pl.N, 256), 256, 0, st>>>((const T*)Pl.pos_tree.p, (const T*)d_q, Pl.perm.p, (T4*)Pl.pq.p, Pl.src_slot.p,
                                                     sizeof(T) == 4 ? Pl.srcg.p : nullptr, Pl.N);
    FMM_CUDA_CHECK(cudaGetLastError());
    dispatch_p2m_l2p<T>(Pl, false, nullptr, nullptr, st, lo, hi);
    FMM_CUDA_CHECK(cudaGetLastError());
}

template <typename T>
void shard_downward_t(const Plan& Pl, const Plan::Shard& sh, void* d_pot, void* d_field, cudaStream_t st) {
    const int L = Pl.L;
    FMM_CUDA_CHECK(cudaMemsetAsync(Pl.Lc.p, 0, Pl.Lc.n, st));
    if (L > 0) FMM_CUDA_CHECK(cudaMemsetAsync(Pl.Mc.p, 0, (size_t)Pl.level_off[L] * Pl.Kp * sizeof(T), st));
    for (int l = L; l > Pl.top_level; --l) xlate_fast_launch(Pl, 0, l, st);              // M2M: every box (redundant on every shard)
    for (int l = 0; l <= L; ++l)
        if (sh.e1[l] > sh.e0[l]) xlate_fast_launch(Pl, 1, 0, st, sh.e0[l], sh.e1[l]);   // M2L: targets of this shard on level l
    for (int l = Pl.top_level + 1; l <= L; ++l)
        if (sh.box_hi[l] > sh.box_lo[l]) xlate_fast_launch(Pl, 2, l, st, sh.box_lo[l], sh.box_hi[l]);  // L2L into its boxes
    if (sizeof(T) == 4) p2p_fast_launch(Pl, st, d_field != nullptr, sh.item0, sh.item1);
    else p2p_fast64_launch(Pl, st, d_field != nullptr, sh.item0, sh.item1);
    FMM_CUDA_CHECK(cudaGetLastError());
    dispatch_p2m_l2p<T>(Pl, true, d_pot, d_field, st, sh.leaf_lo, sh.leaf_hi);
    FMM_CUDA_CHECK(cudaGetLastError());
}

const Plan::Shard& shard_info(const Plan& P, int n_shards, int shard, cudaStream_t st) {
    Plan::Shard& sh = P.shard_cache;
    if (sh.n_shards == n_shards && sh.shard == shard) return sh;
    const int L = P.L;
    sh.box_lo.assign(L + 1, 0); sh.box_hi.assign(L + 1, 0); sh.e0.assign(L + 1, 0); sh.e1.assign(L + 1, 0);
    for (int l = 0; l <= L; ++l) shard_box_range(L, P.s, n_shards, shard, l, &sh.box_lo[l], &sh.box_hi[l]);
    sh.leaf_lo = sh.box_lo[L]; sh.leaf_hi = sh.box_hi[L];
    std::vector<int64_t> h(2 * (L + 1) + 2, 0);
    for (int l = 0; l <= L; ++l) {
        FMM_CUDA_CHECK(cudaMemcpyAsync(&h[2 * l], P.weak_off.p + P.level_off[l] + sh.box_lo[l], sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(&h[2 * l + 1], P.weak_off.p + P.level_off[l] + sh.box_hi[l], sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    }
    FMM_CUDA_CHECK(cudaMemcpyAsync(&h[2 * L + 2], P.p2p_item_off.p + sh.leaf_lo, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    FMM_CUDA_CHECK(cudaMemcpyAsync(&h[2 * L + 3], P.p2p_item_off.p + sh.leaf_hi, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    for (int l = 0; l <= L; ++l) { sh.e0[l] = h[2 * l]; sh.e1[l] = sh.box_hi[l] > sh.box_lo[l] ? h[2 * l + 1] : h[2 * l]; }
    sh.item0 = h[2 * L + 2]; sh.item1 = h[2 * L + 3];
    sh.n_shards = n_shards; sh.shard = shard;
    return sh;
}

void check_shardable(const Plan& P, int n_shards, int shard) {
    if (n_shards < 1 || shard < 0 || shard >= n_shards) { set_error("shard index out of range"); throw CudaFail{FMM_ERR_INVALID_ARG}; }
    if (P.S) { set_error("sharded evaluate: plans with separate targets are not supported"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
    if (!xlate_fast_available(P.p, P.dtype) || P.m2l_variant != 0) {
        set_error("sharded evaluate needs the specialised kernels (1 <= p <= 12, m2l_variant 0)");
        throw CudaFail{FMM_ERR_UNSUPPORTED};
    }
}

}  // namespace

// level-local box range [b0, b1) that shard `shard` of `n_shards` touches on `level`: its leaves on level L, their ancestors above
void shard_box_range(int L, int s, int n_shards, int shard, int level, int64_t* b0, int64_t* b1) {
    const int64_t n_leaves = (int64_t)1 << (s * L);
    const int64_t lo = n_leaves * shard / n_shards, hi = n_leaves * (shard + 1) / n_shards;
    const int sh = s * (L - level);
    *b0 = lo >> sh;
    *b1 = hi > lo ? ((hi - 1) >> sh) + 1 : (lo >> sh);
}

void run_shard_upward(const Plan& P, int n_shards, int shard, const void* d_q, cudaStream_t st) {
    check_shardable(P, n_shards, shard);
    ensure_constants(P);
    int64_t lo, hi;
    shard_box_range(P.L, P.s, n_shards, shard, P.L, &lo, &hi);
    if (P.dtype == FMM_F32) shard_upward_t<float>(P, lo, hi, d_q, st);
    else shard_upward_t<double>(P, lo, hi, d_q, st);
}

void run_shard_downward(const Plan& P, int n_shards, int shard, void* d_pot, void* d_field, cudaStream_t st) {
    check_shardable(P, n_shards, shard);
    ensure_constants(P);
    const Plan::Shard& sh = shard_info(P, n_shards, shard, st);
    if (P.dtype == FMM_F32) shard_downward_t<float>(P, sh, d_pot, d_field, st);
    else shard_downward_t<double>(P, sh, d_pot, d_field, st);
}

namespace {
}  // namespace

int64_t evaluate_launches(const Plan& P) {
    if (P.S) return 5 + (int64_t)P.S->L + (int64_t)P.L + (P.n_weak > 0 ? 1 : 0);  // 2 permutes, P2M, P2P, L2P + M2M/L2L levels + M2L
    const bool fast = P.m2l_variant != 1 && xlate_fast_available(P.p, P.dtype);
    const int64_t w_leaf = (int64_t)P.weak_level_off.size() > P.L ? P.weak_level_off[P.L] : 0;
    int64_t m2l = P.n_weak > 0 ? 1 : 0;
    if (fast && !P.serial && P.L > 0 && w_leaf > 0 && w_leaf < P.n_weak) m2l = 2;  // leaf level and upper levels on two streams
    return 4 + 2 * (int64_t)(P.L - P.top_level) + m2l;  // permute, P2M, P2P, L2P(+finalize) + M2M/L2L per level below top_level + M2L
}

static void run_plain(const Plan& P, const void* d_q, void* d_pot, void* d_field, cudaStream_t st, cudaEvent_t* ev, const void* d_dip) {
    if (P.S) {
        if (P.dtype == FMM_F32) run_st<float>(P, d_q, d_pot, d_field, st, ev, d_dip);
        else run_st<double>(P, d_q, d_pot, d_field, st, ev, d_dip);
    } else if (P.dtype == FMM_F32) run_t<float>(P, d_q, d_pot, d_field, st, ev, d_dip);
    else run_t<double>(P, d_q, d_pot, d_field, st, ev, d_dip);
}

// One evaluate = about 10 + 2 L launches on three streams; below N ~ 1e5 the host cannot issue them as fast as the device retires
// them.  The second evaluate with the same caller pointers is therefore captured (on the plan's own stream: the caller's may be
// the legacy stream, which cannot be captured) and every later one is a single cudaGraphLaunch on the caller's stream.
void run_evaluate(const Plan& P, const void* d_q, void* d_pot, void* d_field, cudaStream_t st, cudaEvent_t* ev, const void* d_dip) {
    ensure_constants(P);
    // above ~5e5 points the device time dwarfs the host's launch cost and the replay measured 2-3 % SLOWER than the stream
    // schedule at N = 1M (the graph starts its branches in another order): large plans keep the plain launches unless told otherwise
    const bool want = P.use_graph == 1 || (P.use_graph == 2 && P.N + (P.S ? P.S->N : 0) < ((int64_t)1 << 19));
    if (ev || !want) { run_plain(P, d_q, d_pot, d_field, st, ev, d_dip); return; }
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        (void)cudaGetLastError();  // the caller is capturing our launches into a graph of their own: the plain schedule is capturable
        run_plain(P, d_q, d_pot, d_field, st, nullptr, d_dip);
        return;
    }
    const uint64_t stamp = (P.epoch << 8) | ((uint64_t)P.m2l_variant << 2) | (P.serial ? 2u : 0u) | (P.deterministic ? 1u : 0u);
    Plan::EvalGraph* g = nullptr;
    for (Plan::EvalGraph& c : P.graphs)
        if (c.seen > 0 && c.q == d_q && c.pot == d_pot && c.fld == d_field && c.dip == d_dip && c.stamp == stamp) { g = &c; break; }
    if (g && g->exec) { FMM_CUDA_CHECK(cudaGraphLaunch(g->exec, st)); return; }
    if (!g) {
        g = &P.graphs[P.graph_next];
        P.graph_next = (P.graph_next + 1) % Plan::N_GRAPHS;
        if (g->exec) {
            FMM_CUDA_CHECK(cudaDeviceSynchronize());  // rare: a fifth set of pointers evicts a graph that may still be running
            cudaGraphExecDestroy(g->exec);
        }
        *g = Plan::EvalGraph();
        g->q = d_q; g->pot = d_pot; g->fld = d_field; g->dip = d_dip; g->stamp = stamp;
    }
    if (g->seen++ == 0) { run_plain(P, d_q, d_pot, d_field, st, nullptr, d_dip); return; }
    if (!P.s_cap) FMM_CUDA_CHECK(cudaStreamCreateWithFlags(&P.s_cap, cudaStreamNonBlocking));
    auto give_up = [&]() {
        (void)cudaGetLastError();
        P.use_graph = 0;
        run_plain(P, d_q, d_pot, d_field, st, nullptr, d_dip);
    };
    if (cudaStreamBeginCapture(P.s_cap, cudaStreamCaptureModeRelaxed) != cudaSuccess) { give_up(); return; }
    cudaGraph_t gr = nullptr;
    try {
        run_plain(P, d_q, d_pot, d_field, P.s_cap, nullptr, d_dip);
    } catch (...) {
        cudaStreamEndCapture(P.s_cap, &gr);
        if (gr) cudaGraphDestroy(gr);
        (void)cudaGetLastError();
        P.use_graph = 0;
        throw;
    }
    if (cudaStreamEndCapture(P.s_cap, &gr) != cudaSuccess || !gr) { give_up(); return; }
    const cudaError_t e = cudaGraphInstantiate(&g->exec, gr, 0);
    cudaGraphDestroy(gr);
    if (e != cudaSuccess) { g->exec = nullptr; give_up(); return; }
    FMM_CUDA_CHECK(cudaGraphLaunch(g->exec, st));
}

// ------------------------------------------------------------------------------------------------ leaf multipoles without allocation
// fmm_leaf_multipoles_noalloc (include/fmm.h): permute + P2M (eq. (13)) of all leaves with the intermediate array of
// the pair -- the particles in tree order packed as (x, y, z, q), which the evaluate keeps in Plan::pq -- in STATIC device memory,
// and the rows written straight into the caller's buffer.  For callers that must not reach cudaMalloc (stream capture, serving
// loops): no allocation here, and nothing of the plan is written, so the call may run beside an evaluate of the same plan.
//
// g_noalloc_pq is a file-scope device array: every GPU that loads the library holds its NOALLOC_BYTES until the process exits.
// In HOST code its name is only a stand-in for the symbol -- never a device address: the address a kernel may be given comes from
// cudaGetSymbolAddress, asked once per device with that device current (noalloc_scratch below).  All calls on a device share the
// array and it keeps the last call's contents: permute_k overwrites records [0, N) and p2m_k reads no others, so nothing has to
// be cleared, but two calls that overlap on the GPU (different streams) race on it.
namespace {

constexpr size_t NOALLOC_BYTES = (size_t)FMM_NOALLOC_MAX_BYTES;
static __device__ __align__(256) unsigned char g_noalloc_pq[NOALLOC_BYTES];

std::mutex g_noalloc_mu;
void* g_noalloc_ptr[MAX_DEVICES] = {};

void* noalloc_scratch(int dev) {
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (dev < 0 || dev >= MAX_DEVICES) { set_error("device ordinal out of range"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
    if (!g_noalloc_ptr[dev]) {
        if (current_device() != dev) { set_error("noalloc scratch: not the current device"); throw CudaFail{FMM_ERR_INVALID_ARG}; }
        void* ptr = nullptr;
        FMM_CUDA_CHECK(cudaGetSymbolAddress(&ptr, g_noalloc_pq));
        g_noalloc_ptr[dev] = ptr;
    }
    return g_noalloc_ptr[dev];
}

template <typename T, int P>
void launch_p2m_to(const Plan& Pl, const void* pq, T* rows_base, cudaStream_t st) {
    using T4 = typename V4<T>::type;
    const int64_t leaf0 = Pl.level_off[Pl.L], nl = Pl.n_leaves;
    if constexpr (sizeof(T) == 4 && P <= 8) {  // the same choice of instantiation as launch_p2m_l2p
        if (Pl.max_leaf <= 16) {
            p2m_k<T, P, 16><<<nblocks(nl, WARPS_PER_BLOCK * 2), WARPS_PER_BLOCK * 32, 0, st>>>((const T4*)pq, Pl.box_start.p, Pl.box_count.p, Pl.box_ctr.p,
                                                                                             (const T*)Pl.box_scale.p, leaf0, nl, Pl.Kp, rows_base);
            return;
        }
    }
    p2m_k<T, P, 32><<<nblocks(nl, WARPS_PER_BLOCK), WARPS_PER_BLOCK * 32, 0, st>>>((const T4*)pq, Pl.box_start.p, Pl.box_count.p, Pl.box_ctr.p,
                                                                                  (const T*)Pl.box_scale.p, leaf0, nl, Pl.Kp, rows_base);
}

template <typename T>
void leaf_multipoles_noalloc_t(const Plan& Pl, const void* d_q, void* d_rows, void* scratch, cudaStream_t st) {
    using T4 = typename V4<T>::type;
    // rows of the leaves only: p2m_k addresses row g of a whole-tree array, so hand it the base that puts leaf 0 at d_rows
    T* rows_base = (T*)d_rows - (int64_t)Pl.level_off[Pl.L] * Pl.Kp;
    FMM_CUDA_CHECK(cudaMemsetAsync(d_rows, 0, (size_t)Pl.n_leaves * Pl.Kp * sizeof(T), st));  // the padding of a row (K..Kp) is zero
    permute_k<T><<<nblocks(Pl.N, 256), 256, 0, st>>>((const T*)Pl.pos_tree.p, (const T*)d_q, Pl.perm.p, (T4*)scratch, nullptr, nullptr, Pl.N);
    FMM_CUDA_CHECK(cudaGetLastError());
    switch (Pl.p) {
#define FMM_CASE(PP) case PP: launch_p2m_to<T, PP>(Pl, scratch, rows_base, st); break;
        FMM_CASE(0) FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
        FMM_CASE(9) FMM_CASE(10) FMM_CASE(11) FMM_CASE(12) FMM_CASE(13) FMM_CASE(14) FMM_CASE(15) FMM_CASE(16)
#undef FMM_CASE
    }
    FMM_CUDA_CHECK(cudaGetLastError());
}

}  // namespace

int64_t noalloc_max_particles(fmm_dtype dt) { return (int64_t)(NOALLOC_BYTES / (4 * (dt == FMM_F32 ? 4 : 8))); }

void run_leaf_multipoles_noalloc(const Plan& P, const void* d_q, void* d_rows, cudaStream_t st) {
    if (P.N > noalloc_max_particles(P.dtype)) {
        set_error("fmm_leaf_multipoles_noalloc: " + std::to_string((long long)P.N) + " particles need " +
                  std::to_string((long long)P.N * 4 * (P.dtype == FMM_F32 ? 4 : 8)) + " bytes of scratch, the static array holds FMM_NOALLOC_MAX_BYTES = " +
                  std::to_string((long long)NOALLOC_BYTES) + " (at most " + std::to_string((long long)noalloc_max_particles(P.dtype)) + " particles of this dtype)");
        throw CudaFail{FMM_ERR_UNSUPPORTED};
    }
    ensure_constants(P);                        // once per device: the g_n^m table in constant memory (a copy, no allocation)
    void* scratch = noalloc_scratch(P.device);  // once per device: cudaGetSymbolAddress
    if (P.dtype == FMM_F32) leaf_multipoles_noalloc_t<float>(P, d_q, d_rows, scratch, st);
    else leaf_multipoles_noalloc_t<double>(P, d_q, d_rows, scratch, st);
}

}  // namespace fmm
