// xlate_smem.cuh -- (instantiated by xlate_smem.cu)
// translation kernels (M2M a5, M2L a6, L2L a7) for fp64 and orders 9 <= p <= 12: ONE THREAD PER TRANSLATION like
// xlate_fast.cu, but the state vector (K = (p+1)^2 = 100..169 doubles) no longer fits the register file, so it lives in
// shared memory, one column per translation, and only the piece an operator step works on is in registers:
//   * the rotations are block diagonal in the degree n: a pass loads one degree (2n+1 <= 25 values), rotates it about z and / or
//     applies the constant matrix, and stores it back;
//   * the z-shift (App. B.3) couples equal orders m only: it loads one order (p+1-|m| values) at a time.
// (fp32 keeps the state in registers up to p = 12 -- 169 + 50 of 255 registers -- and does not use these kernels any more.)
// Same operator, tables and building blocks as the register kernels (xlate_reg.cuh / rot_tables.cuh: the Q Z form with the constant
// matrices as materialised constants, structural zeros free, symmetric pairs sharing one constant).
// In the M2L TWO WARPS SHARE THE 32 COLUMNS OF A BATCH (FMM_SMEM_ROLES = 2): 1352 bytes of state per translation allow only 160
// translations per SM at p = 12, i.e. one warp per scheduler if every translation has one thread; with the passes split between two
// warps -- rotations by degree, shift by order, a CTA barrier where the ownership changes -- the same shared memory feeds two warps
// per scheduler.  Shared layout sm[idx][column] with row stride 33: a thread's own accesses (fixed idx, consecutive columns) and the
// cooperative row copies / run sums (fixed column, consecutive idx) are both conflict-free.
// History (N = 1M uniform cube, fp64 M2L, B200, ms at p = 9 / 10 / 11 / 12): round 1's straight-line B form (three passes over the state,
// 100+ KB of code at p = 12) 3.06 / 5.34 / 7.88 / 14.17; Q Z trips 3.80 / 5.67 / 7.37 / 11.30; trips with two roles 3.56 / 4.82 / 7.76 /
// 9.95; + symmetric constants 3.22 / 4.06 / 6.64 / 8.63 (8.57 with the other kernels' one-warp CTAs beside it); + the two roles paired step by
// step (two degrees per step; +m and -m of the shift at the same time on the same code) 3.06 / 3.76 / 6.17 / 7.86 (this file).
#pragma once
#include "xlate_reg.cuh"

#ifndef FMM_SMEM_ROLES
#define FMM_SMEM_ROLES 2
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
template <int SYNC>  // 2: __syncthreads, 1: compiler fence, 0: nothing (the compiler may overlap neighbouring blocks)
__device__ __forceinline__ void meet() {
    if constexpr (SYNC == 2) __syncthreads();
    else if constexpr (SYNC == 1) fence_block();
}

// state element idx of this thread: col[idx * LD]
// R = 2: two warps share the 32 columns of a batch and split every pass between them -- the rotations by degree, the z-shift by
// order (+m / -m) -- with a CTA barrier where the ownership changes (before and after the shift).  The state of a
// translation stays one column of shared memory; what doubles is the number of warps that work on it.
template <int R>
__device__ __forceinline__ void handover() {
    if constexpr (R > 1) __syncthreads();
}

// ------------------------------------------------------------------------------------------------------------------------
// The operator in the "Q Z loop" form of xlate_reg.cuh (one constant matrix Q_n = polar rotation by pi/2 between azimuthal
// rotations):   Z(pi/2 - phi) Q Z(pi - theta) Q  [(-1)^m S]  Q Z(theta + pi) Q Z(phi + pi/2)
// as SIX TRIPS OF A RUN-TIME LOOP over one copy of "load a degree, rotate it about z, apply Q_n, store it":
//     t = 0: Z(phi + pi/2), Q    1: Z(theta + pi), Q    2: the z-shift    3: Q    4: Z(pi - theta), Q    5: Z(pi/2 - phi)
// A straight-line form holds eight copies of the constant-matrix code (round 1: 100+ KB of SASS at p = 12, far beyond the 32 KB
// instruction cache of an SM); this form holds one, and the z-shift -- whose weights are the same for the orders +m and -m --
// runs its code twice per |m| with a run-time offset into the column (state in shared memory is addressable, registers are
// not).  Cost: six shared-memory round trips of the state instead of three.
template <typename T, int P, int KIND, int am, bool NEG, bool HSYM, int CNT>
__device__ __forceinline__ void shift_order(T (&w)[CNT], const T (&pw1)[P + 1], const T (&pw2)[P + 1], T rinv) {
    // w[k - am], k = am..P: one order of the state (already scaled by x2^k for M2M / M2L); NEG: times (-1)^m = -1
    if constexpr (KIND == 1) {
        T t[CNT];
        if constexpr (HSYM) {  // w scaled by (-x2)^k: the matrix left, (-1)^m X(n, k), is symmetric (xlate_reg.cuh shift_signed)
            sfor<CNT>([&](auto ni) { t[decltype(ni)::value] = T(0); });
            sfor<CNT>([&](auto ni) {
                constexpr int n = am + decltype(ni)::value;
                sfor<CNT - decltype(ni)::value>([&](auto dk) {
                    constexpr int k = n + decltype(dk)::value;
                    constexpr double b = ((k & 1) ? -1.0 : 1.0) * ct::kTab.H[am][n][k];
                    const T c = T(b);
                    t[n - am] = fma(c, w[k - am], t[n - am]);
                    if constexpr (k != n) t[k - am] = fma(c, w[n - am], t[k - am]);
                });
            });
            sfor<CNT>([&](auto ni) { w[decltype(ni)::value] = t[decltype(ni)::value] * (pw1[am + decltype(ni)::value] * rinv); });
        } else {
            sfor<CNT>([&](auto ni) {
                constexpr int n = am + decltype(ni)::value;
                T acc = h_coef<T, am, n, am, NEG>() * w[0];
                sfor<CNT - 1>([&](auto ki) {
                    constexpr int k = am + 1 + decltype(ki)::value;
                    acc = fma(h_coef<T, am, n, k, NEG>(), w[k - am], acc);
                });
                t[decltype(ni)::value] = acc * (pw1[n] * rinv);
            });
            sfor<CNT>([&](auto ni) { w[decltype(ni)::value] = t[decltype(ni)::value]; });
        }
    } else if constexpr (KIND == 0) {
        sfor<CNT>([&](auto ni) {  // in place, n descending
            constexpr int n = P - decltype(ni)::value;
            T acc = NEG ? T(0) - w[n - am] : w[n - am];  // A[m][n][n] = 1
            sfor<n - am>([&](auto ki) {
                constexpr int k = am + decltype(ki)::value;
                acc = fma(a_coef<T, am, n, k, NEG>() * pw1[n - k], w[k - am], acc);
            });
            w[n - am] = acc;
        });
    } else {
        sfor<CNT>([&](auto ni) {  // in place, n ascending
            constexpr int n = am + decltype(ni)::value;
            T acc = w[n - am];
            sfor<P - n>([&](auto ki) {
                constexpr int k = n + 1 + decltype(ki)::value;
                acc = fma(a_coef<T, am, k, n, false>() * pw1[k - n], w[k - am], acc);
            });
            w[n - am] = acc * (NEG ? T(0) - pw2[n] : pw2[n]);
        });
    }
}

template <typename T, int P, int KIND, int LD, int SYNC, int R = 1>
__device__ __forceinline__ void translate_trips(T* __restrict__ col, T bx, T by, T bz, T a_old, T a_new, int role = 0) {
    constexpr int P1 = P + 1;
    // fp64: every "Z(a), then Q" is run as "Z(a + pi), then the symmetric Q D" (q_from_to FORM 1), the lone Q of trip 3 takes its D
    // from the (-1)^m of the shift, which then is the plain shift
    constexpr bool SYM = sizeof(T) == 8;
    T ct_, st_, cp_, sp_, rinv, x1, x2;
    xlate_geometry<T, KIND>(bx, by, bz, a_old, a_new, ct_, st_, cp_, sp_, rinv, x1, x2);
#pragma unroll 1
    for (int t = 0; t < 6; ++t) {
        if (t == 2) {
            T pw1[P1], pw2[P1];
            pw1[0] = pw2[0] = T(1);
            sfor<P>([&](auto jc) {
                pw1[decltype(jc)::value + 1] = pw1[decltype(jc)::value] * x1;
                pw2[decltype(jc)::value + 1] = pw2[decltype(jc)::value] * ((SYM && KIND == 1) ? T(0) - x2 : x2);  // M2L, symmetric shift: (-x2)^k
            });
            handover<R>();  // the rotations were split by degree, the shift is split by order
            sfor<P1>([&](auto mi) {
                constexpr int am = decltype(mi)::value, cnt = P - am + 1;
                constexpr bool NEG = !SYM && (am & 1) != 0;
                // one role: order +am, then -am (same weights, same code); two roles: one of the two orders each, at the same time
                const int sg0 = R == 1 ? 0 : ((role + am) & 1), sg1 = R == 1 ? (am ? 2 : 1) : ((am || sg0 == 0) ? sg0 + 1 : sg0);
#pragma unroll 1
                for (int sg = sg0; sg < sg1; ++sg) {
                    T* cm = col + (sg ? -am : am) * LD;
                    T w[cnt];
                    sfor<cnt>([&](auto ki) {
                        constexpr int k = am + decltype(ki)::value;
                        w[decltype(ki)::value] = cm[(k * k + k) * LD];
                        if constexpr (KIND != 2 && k > 0) w[decltype(ki)::value] *= pw2[k];
                    });
                    shift_order<T, P, KIND, am, NEG, (SYM && KIND == 1)>(w, pw1, pw2, rinv);
                    sfor<cnt>([&](auto ki) {
                        constexpr int k = am + decltype(ki)::value;
                        cm[(k * k + k) * LD] = w[decltype(ki)::value];
                    });
                    if constexpr (R == 1) meet<SYNC>();
                }
                if constexpr (R > 1) meet<SYNC>();  // outside the loop: both roles pass here once per |m|
            });
            handover<R>();
            continue;
        }
        const bool doZ = t != 3, doQ = t != 5;
        T c[P1], s[P1];
        if (doZ) {
            T c1, s1;
            if constexpr (SYM) {  // t = 0: phi + 3 pi/2, 1: theta, 4: -theta, 5: pi/2 - phi
                c1 = (t == 0 || t == 5) ? sp_ : ct_;
                s1 = t == 0 ? T(0) - cp_ : (t == 1 ? st_ : (t == 4 ? T(0) - st_ : cp_));
            } else {
                qz_angle<T>(t < 2 ? t : t - 2, ct_, st_, cp_, sp_, c1, s1);  // t = 4 -> pi - theta (2), t = 5 -> pi/2 - phi (3); t = 3 unused
            }
            trig_table<T, P1>(c1, s1, c, s);
        }
        auto rotate_degree = [&](auto nc) {
            constexpr int n = decltype(nc)::value, w = 2 * n + 1;
            if constexpr (n >= 1 && n <= P) {
                T v[w];
                sfor<w>([&](auto ic) { v[decltype(ic)::value] = col[(n * n + decltype(ic)::value) * LD]; });
                if (doZ) az_from_to<T, n, 0, 0>(v, v, c, s);
                if (doQ) {
                    T tt[w];
                    q_from_to<T, n, 0, 0, q_form<T>(1)>(v, tt);
                    sfor<w>([&](auto ic) { col[(n * n + decltype(ic)::value) * LD] = tt[decltype(ic)::value]; });
                } else {
                    sfor<w>([&](auto ic) { col[(n * n + decltype(ic)::value) * LD] = v[decltype(ic)::value]; });
                }
            }
        };
        if constexpr (R == 1) {
            sfor<P>([&](auto nc) {
                rotate_degree(std::integral_constant<int, decltype(nc)::value + 1>{});
                meet<SYNC>();
            });
        } else {
            // two roles: step k pairs the degrees P - 4 (k / 2) - {0, 3} (role 0) and P - 4 (k / 2) - {1, 2} (role 1): the sums of
            // (2n+1)^2 of the two roles agree to 4 %, and both roles pass the same number of meeting points
            sfor<(P + 1) / 2>([&](auto kc) {
                constexpr int k = decltype(kc)::value, base = P - 4 * (k / 2);
                if (role == 0) rotate_degree(std::integral_constant<int, base - ((k & 1) ? 3 : 0)>{});
                else rotate_degree(std::integral_constant<int, base - ((k & 1) ? 2 : 1)>{});
                meet<SYNC>();
            });
        }
    }
}

// NT threads = NT / R columns (translations) x R roles; MT: what meet<> does after every block (KIND 1 only)
template <typename T, int P, int KIND, int NT, int MT = 2, int R = 1>
__global__ void __launch_bounds__(NT) xlate_smem_k(SArgs a) {
    constexpr int K = (P + 1) * (P + 1), Kp = (K + 3) & ~3, NC = NT / R, LD = NC + 1, NJ = (K + 31) / 32;
    static_assert(NC % 32 == 0 && (R == 1 || R == 2), "columns come in warps; one or two roles");
    extern __shared__ __align__(16) unsigned char smraw[];
    T* sm = reinterpret_cast<T*>(smraw);
    const int lane = threadIdx.x & 31, cw = (threadIdx.x % NC) >> 5, role = threadIdx.x / NC;  // role is uniform in a warp
    const int64_t e = (int64_t)blockIdx.x * NC + threadIdx.x % NC;
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
    constexpr int MEET = KIND == 1 ? MT : 1;
    constexpr bool ALL = MEET == 2 || R > 1;  // every lane walks the operator code (CTA barriers inside)
    const unsigned vmask = __ballot_sync(0xffffffffu, gs >= 0);
    if (!ALL && vmask == 0) return;  // warps are independent (only __syncwarp below) unless they meet at CTA barriers

    // stage in: the source rows of the warp's 32 translations, each read coalesced by a whole warp (R = 2: half of the rows each)
    const T* in = reinterpret_cast<const T*>(a.in);
    T* wcol = sm + cw * 32;
    for (int r = role * (32 / R); r < (role + 1) * (32 / R); ++r) {
        const int g = __shfl_sync(0xffffffffu, gs, r);
        if (g < 0) continue;
        const T* row = in + (int64_t)g * Kp;
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (lane + 32 * j < K) wcol[(lane + 32 * j) * LD + r] = row[lane + 32 * j];
    }
    if constexpr (R > 1) __syncthreads();
    else __syncwarp();
    if (ALL || gs >= 0) {
        const int gs_ = gs >= 0 ? gs : 0, gt_ = gt >= 0 ? gt : 0;
        const T* sc = reinterpret_cast<const T*>(a.scale);
        const T* scs = reinterpret_cast<const T*>(a.scale_s);
        const T bx = (T)(a.ctr_s[3 * (int64_t)gs_] - a.ctr[3 * (int64_t)gt_]);
        const T by = (T)(a.ctr_s[3 * (int64_t)gs_ + 1] - a.ctr[3 * (int64_t)gt_ + 1]);
        const T bz = (T)(a.ctr_s[3 * (int64_t)gs_ + 2] - a.ctr[3 * (int64_t)gt_ + 2]);
        translate_trips<T, P, KIND, LD, MEET, R>(wcol + lane, bx, by, bz, scs[gs_], sc[gt_], role);
    }
    if constexpr (R > 1) __syncthreads();
    else __syncwarp();

    // sum runs of equal targets (lists are sorted by target), one atomicAdd per coefficient and run (R = 2: every other chunk of 32)
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
                if ((R == 1 || (j & 1) == role) && lane + 32 * j < K) acc[j] += wcol[(lane + 32 * j) * LD + r];
        }
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if ((R == 1 || (j & 1) == role) && lane + 32 * j < K) atomicAdd(out + (int64_t)t * Kp + lane + 32 * j, acc[j]);
    }
}

template <typename T, int P, int KIND>
void launch(const SArgs& a, cudaStream_t st) {
    constexpr int K = (P + 1) * (P + 1);
    // M2L: 32 translations per CTA, two warps share them (R = 2) -- twice the warps for the same shared memory; M2M / L2L: 64 per CTA
    // Measured (fp64 M2L, N = 1M, p = 9 / 10 / 11 / 12): 32 columns per CTA, no barrier inside a pass 3.06 / 3.76 / 6.17 / 7.86 ms; ONE CTA of
    // 160 columns x 2 roles per SM whose ten warps meet at a barrier after every block (they walk the code together) 4.78 / 5.51 / 6.28 / 7.64 ms
    constexpr int R = KIND == 1 ? FMM_SMEM_ROLES : 1, NT = KIND == 1 ? 32 * R : 64, MT = 1;
    constexpr size_t smem = (size_t)K * (NT / R + 1) * sizeof(T);
    static AttrOnce once;
    once.ensure(a.device, [&] { FMM_CUDA_CHECK(cudaFuncSetAttribute(xlate_smem_k<T, P, KIND, NT, MT, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); });
    const unsigned grid = (unsigned)((a.n + NT / R - 1) / (NT / R));
    xlate_smem_k<T, P, KIND, NT, MT, R><<<grid, NT, smem, st>>>(a);
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
