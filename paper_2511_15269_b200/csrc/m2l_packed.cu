// m2l_packed.cu -- fp32 M2L (a6), TWO weak pairs per thread in packed f32x2 arithmetic.
//
// Same operator as xlate_fast.cu KIND 1 (App. B):
//     D_t += Z(-phi) B Z(-theta) B^T  [z-shift M2L, PAPER.md:458]  B Z(theta) B^T Z(phi)  C_s ,   b = c_s - c_t  (reading G3)
// but every thread carries the state vectors of two independent interactions in the two halves of 64-bit register pairs
// and runs the fully unrolled operator once with FMUL2 / FFMA2 (sm_100), whose constant operand is a 32-bit immediate
// broadcast to both halves.  One instruction stream therefore serves 64 interactions per warp: the issue slots, the
// instruction fetches and the load/store/reduction overhead per interaction halve, and the FP32 pipe (which executes a
// packed instruction in two passes) becomes the only limiter.
//
// Register budget: 84 packed state values (168 registers) + one cos/sin table (18 packed) or one block of B temporaries
// (17 packed) at a time; the four trig tables are regenerated when needed (8 packed FMAs each) instead of kept alive.
//
// A warp owns 64 consecutive weak pairs (sorted by target); lane l holds pairs l (low half) and 32 + l (high half).
// Source rows arrive in shared memory by TMA bulk copies (one per run of consecutive source ids; row stride an odd number
// of 16-byte units, so the per-lane LDS.128 are conflict-free); the 64 result rows are summed over runs of equal targets
// and added to D with one atomicAdd per coefficient and run.
#include "tma.cuh"
#include "xlate_reg.cuh"

namespace fmm {
namespace {

using namespace xr;


template <int P>
struct PGeo {
    static constexpr int K = (P + 1) * (P + 1);
    static constexpr int Kp = (K + 3) & ~3;
    static constexpr int CH = Kp / 4;                   // 16-byte chunks per row
    static constexpr int KSB = (CH & 1) ? CH : CH + 1;  // shared row stride in 16-byte units (odd)
    static constexpr int KV = CH * 4;
    static constexpr int NJ = (K + 31) / 32;
    static constexpr size_t SMEM_WARP = (size_t)64 * KSB * 16 + 16;  // 64 rows + one mbarrier
};

struct PairGeo {
    float ct, st, cp, sp, x1, x2, rinv;
};

// spherical angles of b = c_s - c_t and the length-scale ratios (a_t / r, a_s / r); centres are fp64 (reading T6)
__device__ __forceinline__ PairGeo pair_geometry(const double* __restrict__ ctr, const float* __restrict__ scale, int gs, int gt) {
    const float bx = (float)(ctr[3 * (int64_t)gs] - ctr[3 * (int64_t)gt]);
    const float by = (float)(ctr[3 * (int64_t)gs + 1] - ctr[3 * (int64_t)gt + 1]);
    const float bz = (float)(ctr[3 * (int64_t)gs + 2] - ctr[3 * (int64_t)gt + 2]);
    const float rxy2 = bx * bx + by * by;
    const float r2 = rxy2 + bz * bz;
    const float r = sqrtf(r2), rxy = sqrtf(rxy2);
    PairGeo g;
    g.rinv = r > 0.f ? 1.f / r : 0.f;
    const float rxyinv = rxy > 0.f ? 1.f / rxy : 0.f;
    g.ct = r > 0.f ? bz * g.rinv : 1.f;
    g.st = rxy * g.rinv;
    g.cp = rxy > 0.f ? bx * rxyinv : 1.f;  // reading S7: phi := 0 on the z axis
    g.sp = by * rxyinv;
    g.x1 = scale[gt] * g.rinv;
    g.x2 = scale[gs] * g.rinv;
    return g;
}

template <int P, int SG, int KV>
__device__ __forceinline__ void az_all(f2 (&v)[KV], f2 c1, f2 s1) {
    f2 c[P + 1], s[P + 1];
    trig_table<f2, P + 1>(c1, s1, c, s);
    sfor<P>([&](auto nc) { apply_az<f2, decltype(nc)::value + 1, SG>(v, c, s); });
}
template <int P, bool TR, int KV>
__device__ __forceinline__ void B_all(f2 (&v)[KV]) {
    sfor<P>([&](auto nc) { apply_B<f2, decltype(nc)::value + 1, TR>(v); });
}

// SYNC: the warps of the CTA meet at a barrier after every phase (lockstep => shared instruction-cache lines)
template <int P, bool SYNC, int KV>
__device__ __forceinline__ void m2l_pair(f2 (&v)[KV], f2 ct, f2 st, f2 cp, f2 sp, f2 x1, f2 x2, f2 rinv) {
    auto sync = [] { if constexpr (SYNC) __syncthreads(); };
    constexpr int P1 = P + 1;
    // source length scale: degree k carries (a_s / r)^k
    {
        f2 pw = x2;
        sfor<P>([&](auto nc) {
            constexpr int n = decltype(nc)::value + 1;
            sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
            if constexpr (n < P) pw *= x2;
        });
    }
    // forward rotation  B Z(theta) B^T Z(phi)  brings b onto +z
    az_all<P, +1>(v, cp, sp);
    sync();
    B_all<P, true>(v);
    sync();
    az_all<P, +1>(v, ct, st);
    B_all<P, false>(v);
    sync();
    // z-shift (App. B.3) in the normalised basis: only equal orders m couple
    sfor<2 * P + 1>([&](auto mi) {
        constexpr int m = decltype(mi)::value - P, am = m < 0 ? -m : m, cnt = P - am + 1;
        f2 t[cnt];
        sfor<cnt>([&](auto ni) {
            constexpr int n = am + decltype(ni)::value;
            constexpr double h0 = ct::kTab.H[am][n][am];
            f2 acc = f2(h0) * v[am * am + am + m];
            sfor<cnt - 1>([&](auto ki) {
                constexpr int k = am + 1 + decltype(ki)::value;
                constexpr double h = ct::kTab.H[am][n][k];
                acc = fma(f2(h), v[k * k + k + m], acc);
            });
            t[decltype(ni)::value] = acc;
        });
        sfor<cnt>([&](auto ni) { v[(am + decltype(ni)::value) * (am + decltype(ni)::value + 1) + m] = t[decltype(ni)::value]; });
    });
    // target length scale: degree n carries (a_t / r)^n / r
    {
        f2 pw = rinv;
        sfor<P1>([&](auto nc) {
            constexpr int n = decltype(nc)::value;
            sfor<2 * n + 1>([&](auto ic) { v[n * n + decltype(ic)::value] *= pw; });
            if constexpr (n < P) pw *= x1;
        });
    }
    // inverse rotation  Z(-phi) B Z(-theta) B^T
    sync();
    B_all<P, true>(v);
    sync();
    az_all<P, -1>(v, ct, st);
    B_all<P, false>(v);
    sync();
    az_all<P, -1>(v, cp, sp);
}

template <int P, int MW, bool SYNC>
__global__ void __launch_bounds__(MW * 32, 8 / MW)
m2l_packed_k(int64_t n, const int32_t* __restrict__ wtgt, const int32_t* __restrict__ wsrc, const double* __restrict__ ctr,
             const float* __restrict__ scale, const float* __restrict__ Mc, float* __restrict__ Lc) {
    using G = PGeo<P>;
    extern __shared__ __align__(16) unsigned char smraw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* wbase = smraw + (size_t)warp * G::SMEM_WARP;
    float4* sm = reinterpret_cast<float4*>(wbase);
    const uint32_t bar = smem_u32(wbase + (size_t)64 * G::KSB * 16);
    int64_t e0 = ((int64_t)blockIdx.x * MW + warp) * 64;
    if constexpr (SYNC) {
        if (e0 >= n) e0 = n;  // idle warps still walk the code (barriers); all their pairs are discarded
    } else {
        if (e0 >= n) return;
    }

    // pairs of this lane: e0 + lane (low half, shared row `lane`) and e0 + 32 + lane (high half, shared row 32 + lane)
    const int64_t eA = e0 + lane, eB = eA + 32;
    int gsA = -1, gtA = -1, gsB = -1, gtB = -1;
    if (eA < n) { gsA = wsrc[eA]; gtA = wtgt[eA]; }
    if (eB < n) { gsB = wsrc[eB]; gtB = wtgt[eB]; }
    if (lane == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncwarp();

    // source rows by TMA bulk copies, one per run of consecutive source ids (see xlate_fast.cu), all on one mbarrier
    constexpr uint32_t ROWB = G::CH * 16;
    auto fetch = [&](int gs, int rowbase) -> int {
        const int gprev = __shfl_up_sync(0xffffffffu, gs, 1);
        const bool head = lane == 0 || gs < 0 || gprev < 0 || gs != gprev + 1 || G::KSB != G::CH;
        const unsigned hm = __ballot_sync(0xffffffffu, head);
        const unsigned above = lane == 31 ? 0u : (hm >> (lane + 1));
        const int len = above ? __ffs(above) : 32 - lane;
        if (head && gs >= 0)
            bulk_g2s(smem_u32(sm + (rowbase + lane) * G::KSB), reinterpret_cast<const char*>(Mc) + (int64_t)gs * ROWB, (uint32_t)len * ROWB, bar);
        return __popc(__ballot_sync(0xffffffffu, gs >= 0));
    };
    const int nA = fetch(gsA, 0), nB = fetch(gsB, 32);
    if (lane == 0) mbar_expect_tx(bar, (uint32_t)(nA + nB) * ROWB);
    // padding pairs compute on whatever their shared rows hold (their results are discarded), with a harmless geometry
    const PairGeo ga = pair_geometry(ctr, scale, gsA >= 0 ? gsA : 0, gsA >= 0 ? gtA : 1);
    const PairGeo gb = pair_geometry(ctr, scale, gsB >= 0 ? gsB : 0, gsB >= 0 ? gtB : 1);
    mbar_wait(bar, 0);

    f2 v[G::KV];
    {
        const float4* rowA = sm + lane * G::KSB;
        const float4* rowB = sm + (32 + lane) * G::KSB;
        sfor<G::CH>([&](auto cc) {
            constexpr int c = decltype(cc)::value;
            const float4 xa = rowA[c], xb = rowB[c];
            v[4 * c] = f2(xa.x, xb.x);
            v[4 * c + 1] = f2(xa.y, xb.y);
            v[4 * c + 2] = f2(xa.z, xb.z);
            v[4 * c + 3] = f2(xa.w, xb.w);
        });
    }
    __syncwarp();  // all rows are in registers: the buffer is reused for the results

    m2l_pair<P, SYNC>(v, f2(ga.ct, gb.ct), f2(ga.st, gb.st), f2(ga.cp, gb.cp), f2(ga.sp, gb.sp), f2(ga.x1, gb.x1), f2(ga.x2, gb.x2),
                f2(ga.rinv, gb.rinv));

    {
        float4* rowA = sm + lane * G::KSB;
        float4* rowB = sm + (32 + lane) * G::KSB;
        sfor<G::CH>([&](auto cc) {
            constexpr int c = decltype(cc)::value;
            rowA[c] = make_float4(v[4 * c].lo(), v[4 * c + 1].lo(), v[4 * c + 2].lo(), v[4 * c + 3].lo());
            rowB[c] = make_float4(v[4 * c].hi(), v[4 * c + 1].hi(), v[4 * c + 2].hi(), v[4 * c + 3].hi());
        });
    }
    __syncwarp();

    // sum runs of equal targets over the 64 rows (the list is sorted by target): run heads by ballots, warp-uniform row
    // loops, one atomicAdd per coefficient and run; lane j owns coefficients j, j+32, j+64
    const float* smT = reinterpret_cast<const float*>(sm);
    constexpr int RS = G::KSB * 4;  // shared row stride in floats
    const int pA = __shfl_up_sync(0xffffffffu, gtA, 1), lastA = __shfl_sync(0xffffffffu, gtA, 31);
    const int pB = __shfl_up_sync(0xffffffffu, gtB, 1);
    const unsigned hA = __ballot_sync(0xffffffffu, lane == 0 || gtA != pA);
    const unsigned hB = __ballot_sync(0xffffffffu, lane == 0 ? gtB != lastA : gtB != pB);
    unsigned long long heads = (unsigned long long)hA | ((unsigned long long)hB << 32);
    while (heads) {
        const int r0 = __ffsll((long long)heads) - 1;
        heads &= heads - 1;
        const int r1 = heads ? __ffsll((long long)heads) - 1 : 64;
        const int t = r0 < 32 ? __shfl_sync(0xffffffffu, gtA, r0) : __shfl_sync(0xffffffffu, gtB, r0 - 32);
        if (t < 0) continue;  // padding pairs
        float acc[G::NJ];
#pragma unroll
        for (int j = 0; j < G::NJ; ++j) acc[j] = 0.f;
#pragma unroll 8
        for (int r = r0; r < r1; ++r) {
#pragma unroll
            for (int j = 0; j < G::NJ; ++j)
                if (lane + 32 * j < G::K) acc[j] += smT[r * RS + lane + 32 * j];
        }
#pragma unroll
        for (int j = 0; j < G::NJ; ++j)
            if (lane + 32 * j < G::K) atomicAdd(Lc + (int64_t)t * G::Kp + lane + 32 * j, acc[j]);
    }
}

template <int P, int MW = 4, bool SYNC = false>
void launch_packed(const Plan& Pl, cudaStream_t st, int64_t e0, int64_t e1) {
    using G = PGeo<P>;
    constexpr size_t smem = (size_t)MW * G::SMEM_WARP;
    static bool attr_set = false;
    if (!attr_set) {
        FMM_CUDA_CHECK(cudaFuncSetAttribute(m2l_packed_k<P, MW, SYNC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    const unsigned grid = (unsigned)((e1 - e0 + MW * 64 - 1) / (MW * 64));
    m2l_packed_k<P, MW, SYNC><<<grid, MW * 32, smem, st>>>(e1 - e0, Pl.weak_tgt.p + e0, Pl.weak_src.p + e0, Pl.box_ctr.p, (const float*)Pl.box_scale.p,
                                                 (const float*)Pl.Mc.p, (float*)Pl.Lc.p);
}

}  // namespace

bool m2l_packed_available(int p, fmm_dtype dt) { return dt == FMM_F32 && p >= 1 && p <= 8; }

void m2l_packed_launch(const Plan& P, cudaStream_t st, int64_t e0, int64_t e1) {
    if (e1 <= e0) return;
    switch (P.p) {
#define FMM_CASE(PP) case PP: launch_packed<PP>(P, st, e0, e1); break;
        FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
#undef FMM_CASE
        default: set_error("no packed M2L kernel for this order"); throw CudaFail{FMM_ERR_UNSUPPORTED};
    }
}

}  // namespace fmm
