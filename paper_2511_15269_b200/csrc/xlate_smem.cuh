// xlate_smem.cuh -- (instantiated per dtype by xlate_smem_f32.cu / xlate_smem_f64.cu, so that the two compile in parallel)
// translation kernels (M2M a5, M2L a6, L2L a7) for orders 9 <= p <= 12, fp32 and fp64: ONE THREAD PER
// TRANSLATION like xlate_fast.cu, but the state vector (K = (p+1)^2 = 100..169 values) no longer fits the register file,
// so it lives in shared memory, one column per thread, and only the piece an operator step works on is in registers:
//   * the rotations Z(phi), B^T, Z(theta), B (and their inverses) are block diagonal in the degree n, so the forward and
//     the inverse rotation load one degree (2n+1 <= 25 values), apply all four factors in registers, and store it back;
//   * the z-shift (App. B.3) couples equal orders m only: it loads one order (p+1-|m| values) at a time.
// Same operator, tables and building blocks as the register kernels (xlate_reg.cuh / rot_tables.cuh: constant matrices
// B_n as immediates, structural zeros free); three shared-memory round trips per coefficient replace the register
// residency.  Shared layout sm[idx][thread] with row stride NT+1: a thread's own accesses (fixed idx, consecutive
// threads) and the cooperative row copies / run sums (fixed thread column, consecutive idx) are both conflict-free.
#pragma once
#include "xlate_reg.cuh"

#ifndef FMM_SMEM_SYNC
#define FMM_SMEM_SYNC 1
#endif

namespace fmm {
namespace {

using namespace xr;

struct SArgs {
    int device;                   // host side only: the plan's device (per-device kernel attributes)
    int64_t first;                // KIND 0 / 2: first child (level-local index) of this launch
    int64_t n;                    // number of translations
    const int32_t *tgt, *src;     // KIND 1: global ids per pair
    int64_t off_parent, off_child;
    int s;
    const int32_t* box_count;
    const double* ctr;            // output side (see XArgs in xlate_fast.cu)
    const void* scale;
    const double* ctr_s;          // input side
    const void* scale_s;
    const void* in;
    void* out;
};

// compiler-only barrier between two blocks: keeps the loads of the next block behind the stores of this one, so that
// only one block (plus the trig / power tables) is live in registers at a time
__device__ __forceinline__ void fence_block() { asm volatile("" ::: "memory"); }
// SYNC: the warps of a CTA meet after every block, so that they walk the (100+ KB, straight-line) code together and share
// instruction-cache lines
template <bool SYNC>
__device__ __forceinline__ void meet() {
    if constexpr (SYNC) __syncthreads();
    else fence_block();
}

// state element idx of this thread: col[idx * LD]
template <typename T, int P, int KIND, int LD, bool SYNC>
__device__ __forceinline__ void translate_blocked(T* __restrict__ col, T bx, T by, T bz, T a_old, T a_new) {
    constexpr int P1 = P + 1, K = P1 * P1;
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

    T v[K];  // only the block in flight is live
    // forward rotation, degree by degree (degree 0 is invariant); M2M / M2L fold the source scaling x2^n in
    {
        T pw = T(1);
        sfor<P>([&](auto nc) {
            constexpr int n = decltype(nc)::value + 1;
            sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] = col[(n * n + decltype(ic)::value) * LD]; });
            if constexpr (KIND != 2) {
                pw *= x2;
                sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
            }
            apply_az<T, n, +1>(v, cph, sph);
            apply_B<T, n, true>(v);
            apply_az<T, n, +1>(v, cth, sth);
            apply_B<T, n, false>(v);
            sfor<2 * n + 1>([&](auto ic) { col[(n * n + decltype(ic)::value) * LD] = v[n * n + decltype(ic)::value]; });
            meet<SYNC>();
        });
    }

    // z-shift, order by order
    T pw1[P1];
    pw1[0] = T(1);
    sfor<P>([&](auto jc) { pw1[decltype(jc)::value + 1] = pw1[decltype(jc)::value] * x1; });
    T pw2[P1];
    pw2[0] = T(1);
    sfor<P>([&](auto jc) { pw2[decltype(jc)::value + 1] = pw2[decltype(jc)::value] * x2; });
    sfor<2 * P + 1>([&](auto mi) {
        constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
        sfor<cnt>([&](auto ki) {
            constexpr int k = am + decltype(ki)::value;
            v[k * k + k + m] = col[(k * k + k + m) * LD];
        });
        if constexpr (KIND == 1) {
            // out[n] = (x1^n / r) sum_k H[|m|][n][k] v[k]   (v already scaled by x2^k)
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
                t[decltype(ni)::value] = acc * (pw1[n] * rinv);
            });
            sfor<cnt>([&](auto ni) {
                constexpr int n = am + decltype(ni)::value;
                col[(n * n + n + m) * LD] = t[decltype(ni)::value];
            });
        } else if constexpr (KIND == 0) {
            // out[n] = sum_{k=|m|..n} A[|m|][n][k] x1^(n-k) v[k]: in place, n descending
            sfor<cnt>([&](auto ni) {
                constexpr int n = P - decltype(ni)::value;
                T acc = v[n * n + n + m];  // A[m][n][n] = 1
                sfor<n - am>([&](auto ki) {
                    constexpr int k = am + decltype(ki)::value;
                    constexpr double aa = ct::kTab.A[am][n][k];
                    acc = fma(T(aa) * pw1[n - k], v[k * k + k + m], acc);
                });
                col[(n * n + n + m) * LD] = acc;
            });
        } else {
            // out[n] = x2^n sum_{k=n..p} A[|m|][k][n] x1^(k-n) v[k]: in place, n ascending
            sfor<cnt>([&](auto ni) {
                constexpr int n = am + decltype(ni)::value;
                T acc = v[n * n + n + m];
                sfor<P - n>([&](auto ki) {
                    constexpr int k = n + 1 + decltype(ki)::value;
                    constexpr double aa = ct::kTab.A[am][k][n];
                    acc = fma(T(aa) * pw1[k - n], v[k * k + k + m], acc);
                });
                col[(n * n + n + m) * LD] = acc * pw2[n];
            });
        }
        meet<SYNC>();
    });

    // inverse rotation
    sfor<P>([&](auto nc) {
        constexpr int n = decltype(nc)::value + 1;
        sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] = col[(n * n + decltype(ic)::value) * LD]; });
        apply_B<T, n, true>(v);
        apply_az<T, n, -1>(v, cth, sth);
        apply_B<T, n, false>(v);
        apply_az<T, n, -1>(v, cph, sph);
        sfor<2 * n + 1>([&](auto ic) { col[(n * n + decltype(ic)::value) * LD] = v[n * n + decltype(ic)::value]; });
        meet<SYNC>();
    });
}

template <typename T, int P, int KIND, int NT>
__global__ void __launch_bounds__(NT) xlate_smem_k(SArgs a) {
    constexpr int K = (P + 1) * (P + 1), Kp = (K + 3) & ~3, LD = NT + 1, NJ = (K + 31) / 32;
    extern __shared__ __align__(16) unsigned char smraw[];
    T* sm = reinterpret_cast<T*>(smraw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t e = (int64_t)blockIdx.x * NT + threadIdx.x;
    int gs = -1, gt = -1;
    if (e < a.n) {
        if constexpr (KIND == 1) { gs = a.src[e]; gt = a.tgt[e]; }
        else {
            const int64_t c = a.first + e;
            const int64_t gc = a.off_child + c, gp = a.off_parent + (c >> a.s);
            if (a.box_count[gc] > 0) {
                if constexpr (KIND == 0) { gs = (int)gc; gt = (int)gp; }
                else { gs = (int)gp; gt = (int)gc; }
            }
        }
    }
    constexpr bool SYNC = KIND == 1 && FMM_SMEM_SYNC;
    const unsigned vmask = __ballot_sync(0xffffffffu, gs >= 0);
    if (!SYNC && vmask == 0) return;  // warps are independent (only __syncwarp below) unless they walk the code in lockstep

    // stage in: the source rows of the warp's 32 translations, each read coalesced by the whole warp
    const T* in = reinterpret_cast<const T*>(a.in);
    T* wcol = sm + warp * 32;
    for (int r = 0; r < 32; ++r) {
        const int g = __shfl_sync(0xffffffffu, gs, r);
        if (g < 0) continue;
        const T* row = in + (int64_t)g * Kp;
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (lane + 32 * j < K) wcol[(lane + 32 * j) * LD + r] = row[lane + 32 * j];
    }
    __syncwarp();
    if (SYNC || gs >= 0) {
        const int gs_ = gs >= 0 ? gs : 0, gt_ = gt >= 0 ? gt : 0;
        const T* sc = reinterpret_cast<const T*>(a.scale);
        const T* scs = reinterpret_cast<const T*>(a.scale_s);
        const T bx = (T)(a.ctr_s[3 * (int64_t)gs_] - a.ctr[3 * (int64_t)gt_]);
        const T by = (T)(a.ctr_s[3 * (int64_t)gs_ + 1] - a.ctr[3 * (int64_t)gt_ + 1]);
        const T bz = (T)(a.ctr_s[3 * (int64_t)gs_ + 2] - a.ctr[3 * (int64_t)gt_ + 2]);
        translate_blocked<T, P, KIND, LD, SYNC>(wcol + lane, bx, by, bz, scs[gs_], sc[gt_]);
    }
    __syncwarp();

    // sum runs of equal targets (lists are sorted by target), one atomicAdd per coefficient and run
    T* out = reinterpret_cast<T*>(a.out);
    const int prev = __shfl_up_sync(0xffffffffu, gt, 1);
    unsigned heads = __ballot_sync(0xffffffffu, lane == 0 || gt != prev);
    while (heads) {
        const int r0 = __ffs(heads) - 1;
        heads &= heads - 1;
        const int r1 = heads ? __ffs(heads) - 1 : 32;
        const int t = __shfl_sync(0xffffffffu, gt, r0);
        if (t < 0) continue;  // padding lanes / empty boxes
        T acc[NJ];
#pragma unroll
        for (int j = 0; j < NJ; ++j) acc[j] = T(0);
        for (int r = r0; r < r1; ++r) {
#pragma unroll
            for (int j = 0; j < NJ; ++j)
                if (lane + 32 * j < K) acc[j] += wcol[(lane + 32 * j) * LD + r];
        }
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (lane + 32 * j < K) atomicAdd(out + (int64_t)t * Kp + lane + 32 * j, acc[j]);
    }
}

template <typename T, int P, int KIND>
void launch(const SArgs& a, cudaStream_t st) {
    constexpr int NT = sizeof(T) == 4 ? 128 : 64;
    constexpr int K = (P + 1) * (P + 1);
    constexpr size_t smem = (size_t)K * (NT + 1) * sizeof(T);
    static AttrOnce once;
    once.ensure(a.device, [&] { FMM_CUDA_CHECK(cudaFuncSetAttribute(xlate_smem_k<T, P, KIND, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); });
    const unsigned grid = (unsigned)((a.n + NT - 1) / NT);
    xlate_smem_k<T, P, KIND, NT><<<grid, NT, smem, st>>>(a);
}

template <typename T, int KIND>
bool dispatch(int p, const SArgs& a, cudaStream_t st) {
    switch (p) {
#define FMM_CASE(PP) case PP: launch<T, PP, KIND>(a, st); return true;
        FMM_CASE(9) FMM_CASE(10) FMM_CASE(11) FMM_CASE(12)
#undef FMM_CASE
        default: return false;
    }
}


template <typename T>
bool smem_launch_t(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    SArgs a{};
    a.device = P.device;
    a.box_count = P.box_count.p;
    a.ctr = a.ctr_s = P.box_ctr.p;
    a.scale = a.scale_s = P.box_scale.p;
    a.s = P.s;
    if (kind == 1) {
        if (e1 < 0) e1 = P.n_weak;
        a.n = e1 - e0;
        a.tgt = P.weak_tgt.p + e0;
        a.src = P.weak_src.p + e0;
        a.in = P.Mc.p;
        a.out = P.Lc.p;
        if (P.S) { a.ctr_s = P.S->box_ctr.p; a.scale_s = P.S->box_scale.p; a.in = P.S->Mc.p; }
    } else {
        a.first = e1 < 0 ? 0 : e0;
        a.n = e1 < 0 ? ((int64_t)1 << (P.s * level)) : e1 - e0;  // children on `level`
        a.off_parent = P.level_off[level - 1];
        a.off_child = P.level_off[level];
        a.in = kind == 0 ? P.Mc.p : P.Lc.p;
        a.out = kind == 0 ? P.Mc.p : P.Lc.p;
    }
    if (a.n <= 0) return true;
    if (kind == 0) return dispatch<T, 0>(P.p, a, st);
    if (kind == 1) return dispatch<T, 1>(P.p, a, st);
    return dispatch<T, 2>(P.p, a, st);
}

}  // namespace
}  // namespace fmm
