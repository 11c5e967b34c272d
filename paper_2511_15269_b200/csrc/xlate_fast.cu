// xlate_fast.cu -- register ("fast") translation kernels: M2M (a5), M2L (a6) and L2L (a7) with ONE THREAD PER TRANSLATION.
// Orders 1..8 in fp32 and fp64, orders 9..12 in fp32 (169 state registers + one degree of temporaries fit the 255-register budget
// at two CTAs of four warps per SM: fp32 p = 12 M2L at N = 1M 2.04 ms against 3.30 ms with the state in shared memory).
//
// The operator is the paper's rotate / shift-along-z / rotate-back (App. B) in the
// normalised, length-scaled representation of tables.cu, where rotations are orthogonal and the polar rotation factors
// through ONE constant matrix Q_n = polar rotation by pi/2 (rot_tables.cuh), applied four times between azimuthal rotations:
//     Z(pi/2 - phi) Q Z(pi - theta) Q  [(-1)^m z-shift]  Q Z(theta + pi) Q Z(phi + pi/2)         (xlate_reg.cuh translate_qz)
// i.e. four azimuthal rotations (4 FP32 instructions per +-m pair), four applications of the constant, 3/4-empty Q (247 MACs each at
// p = 8) and one O(p^3) z-shift (489 MACs at p = 8): about 2.35 k FP32 instructions at p = 8, run as a loop over one copy of the Q code.
//
// Why one thread per translation instead of the paper's / north_star's "one warp per interaction": every step is a
// batch of small, ragged mat-vecs (block sizes 1..2p+1) with a different right-hand side per interaction, which maps
// badly onto 32 lanes (K = 81 is 2.5 warps wide, rows have different lengths).  With one interaction per lane the whole
// warp executes the same fully unrolled instruction stream, all matrix entries are immediates, the state vector lives
// in registers, and there is no shuffle or shared-memory traffic inside the operator.  Shared memory is only the staging
// area: every lane fetches its source row with one TMA bulk copy (cp.async.bulk + mbarrier) and reads it with conflict-free
// LDS.128 (row stride an odd number of 16-byte units); results go back the same way and are summed over runs of equal
// targets (the lists are sorted by target) before one atomicAdd per coefficient and run.
#include "tma.cuh"
#include "xlate_reg.cuh"

// Form of the Q Z loop (xlate_reg.cuh translate_qz), measured on B200 (N = 1M, p = 8, M2L stage): fp32: MODE 0 (A / B trips, no
// register copies) 0.691 ms, MODE 2 (Q in place) 0.700 ms, MODE 1 (one Q copy + identity trip) 0.75 ms; fp64: MODE 2 1.55 ms,
// MODE 0 1.66 ms (255 registers either way; MODE 0 spills a little more).  fp32, p = 9 / 10 / 12: MODE 2 0.92 / 1.17 / 2.04 ms, MODE 0
// 0.95 / 1.35 / 2.04 ms.
template <typename T, int P = 8> constexpr int qz_mode() { return (P > 8 || sizeof(T) == 8) ? 2 : 0; }

namespace fmm {
namespace {

using namespace xr;


template <typename T> struct Vec16;
template <> struct Vec16<float> { using type = float4; static constexpr int E = 4; };
template <> struct Vec16<double> { using type = double2; static constexpr int E = 2; };

template <typename T, int P>
struct Geo {
    static constexpr int K = (P + 1) * (P + 1);
    static constexpr int E = Vec16<T>::E;
    static constexpr int Kp = (K + 3) & ~3;            // row stride of the global coefficient arrays (elements)
    static constexpr int CH = Kp / E;                  // 16-byte chunks per global row
    static constexpr int KSB = (CH & 1) ? CH : CH + 1; // shared row stride in 16-byte units: odd => conflict-free LDS.128
    static constexpr int KV = CH * E;                  // register vector length
    static constexpr int NJ = (K + 31) / 32;
};

struct XArgs {
    int device;                   // host side only: the plan's device (per-device kernel attributes)
    int64_t first;                // KIND 0 / 2: first child (level-local index) of this launch
    int64_t n;                    // number of translations
    const int32_t *tgt, *src;     // KIND 1: global ids per pair
    int64_t off_parent, off_child;
    int s;
    const int32_t* box_count;
    const double* ctr;            // box centres / scales of the hierarchy the OUTPUT boxes belong to
    const void* scale;
    const double* ctr_s;          // ... and of the hierarchy the INPUT boxes belong to (the same arrays unless the M2L joins
    const void* scale_s;          //     a source hierarchy to a separate target hierarchy)
    const void* in;
    void* out;
    const int64_t* woff;          // m2l_row_k: CSR offsets of the weak list by target box
    const float* geo;             // KIND 1, GEO kernels: geometry records of the pairs (m2l_geo_prepare), 1 KB per batch of 32
};

// XW warps per CTA; GEO (fp32 M2L only): target ids and the geometry of every pair (cos / sin of the two angles, 1/r, scale ratios)
// come from records written at plan time (m2l_geo_prepare) -- one coalesced load per word instead of a gather of fp64 centres
// that depends on the ids, and no square roots or divisions in the kernel.
// One warp per CTA (XW = 1): the warps of a CTA never cooperate, and a CTA keeps its registers and shared memory until its slowest
// warp is done -- batches differ (number of target runs in the epilogue, TMA copies in the prologue).  Measured on B200, config 2 M2L:
// 4 warps per CTA 0.695 ms, 2: 0.683 ms, 1: 0.659 ms (config 4, p = 6: 1.60 -> 1.28 ms).  Warps per SM by the register budget:
// fp32 p <= 8: 16 (128 registers), p = 9, 10: 12 (168), fp32 p = 11, 12 and fp64: 8 (255).
template <typename T, int P>
constexpr int xlate_warps_per_sm() { return sizeof(T) == 8 ? 8 : (P > 10 ? 8 : (P > 8 ? 12 : 16)); }
template <typename T, int P, int KIND, int XW, bool GEO>
__global__ void __launch_bounds__(XW * 32, xlate_warps_per_sm<T, P>() / XW) xlate_fast_k(XArgs a) {
    using G = Geo<T, P>;
    using V = typename Vec16<T>::type;
    extern __shared__ __align__(16) unsigned char smraw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    V* sm = reinterpret_cast<V*>(smraw) + (size_t)warp * 32 * G::KSB;
    const int64_t e = ((int64_t)blockIdx.x * XW + warp) * 32 + lane;
    int gs = -1, gt = -1;
    float rec[7];  // GEO: ct, st, cp, sp, 1/r, x1, x2
    if constexpr (GEO) {
        // the record block of this warp's batch: word w of pair `lane` at rec[w * 32 + lane]; padding pairs carry gt = -1
        const float* r = a.geo + (e >> 5) * 256 + lane;
#pragma unroll
        for (int w = 0; w < 7; ++w) rec[w] = r[32 * w];
        if (e < a.n) {  // a launch may cover only a prefix of the segment (sharded evaluate): pairs beyond it are not this launch's
            gt = reinterpret_cast<const int*>(r)[224];
            gs = a.src[e];
        }
    } else if (e < a.n) {
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
    const unsigned vmask = __ballot_sync(0xffffffffu, gs >= 0);
    if (vmask == 0) return;

    // source rows (CH * 16 contiguous bytes each) arrive by TMA bulk copies that complete on one mbarrier per warp, so the
    // whole batch is in flight at once while the geometry is being loaded
    constexpr uint32_t ROWB = G::CH * 16;
    const uint32_t bar = smem_u32(reinterpret_cast<unsigned long long*>(smraw + (size_t)XW * 32 * G::KSB * 16) + warp);
    if (lane == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncwarp();
    // consecutive lanes with consecutive source ids (siblings are numbered consecutively and the lists are sorted) read one
    // contiguous piece of the coefficient array: the first lane of such a run copies the whole run (possible when the shared
    // rows are contiguous too, KSB == CH); a bulk copy is issued by one elected lane at a time, so fewer copies matter
    {
        const int gprev = __shfl_up_sync(0xffffffffu, gs, 1);
        const bool head = lane == 0 || gs < 0 || gprev < 0 || gs != gprev + 1 || G::KSB != G::CH;
        const unsigned hm = __ballot_sync(0xffffffffu, head);
        const unsigned above = lane == 31 ? 0u : (hm >> (lane + 1));
        const int len = above ? __ffs(above) : 32 - lane;
        if (head && gs >= 0)
            bulk_g2s(smem_u32(sm + lane * G::KSB), reinterpret_cast<const char*>(a.in) + (int64_t)gs * ROWB, (uint32_t)len * ROWB, bar);
    }
    if (lane == 0) mbar_expect_tx(bar, (uint32_t)__popc(vmask) * ROWB);
    T bx = T(0), by = T(0), bz = T(1), a_old = T(1), a_new = T(1);
    if (!GEO && gs >= 0) {
        const T* sc = reinterpret_cast<const T*>(a.scale);
        const T* scs = reinterpret_cast<const T*>(a.scale_s);
        bx = (T)(a.ctr_s[3 * (int64_t)gs] - a.ctr[3 * (int64_t)gt]);
        by = (T)(a.ctr_s[3 * (int64_t)gs + 1] - a.ctr[3 * (int64_t)gt + 1]);
        bz = (T)(a.ctr_s[3 * (int64_t)gs + 2] - a.ctr[3 * (int64_t)gt + 2]);
        a_old = scs[gs];
        a_new = sc[gt];
    }
    mbar_wait(bar, 0);

    T v[G::KV];
    V* row = sm + lane * G::KSB;
    if (gs >= 0) {
        sfor<G::CH>([&](auto cc) {
            constexpr int c = decltype(cc)::value;
            const V x = row[c];
            if constexpr (G::E == 4) { v[4 * c] = x.x; v[4 * c + 1] = x.y; v[4 * c + 2] = x.z; v[4 * c + 3] = x.w; }
            else { v[2 * c] = x.x; v[2 * c + 1] = x.y; }
        });
        if constexpr (GEO) translate_qz_geo<T, P, KIND, qz_mode<T, P>()>(v, (T)rec[0], (T)rec[1], (T)rec[2], (T)rec[3], (T)rec[4], (T)rec[5], (T)rec[6]);
        else translate_qz<T, P, KIND, qz_mode<T, P>()>(v, bx, by, bz, a_old, a_new);
        sfor<G::CH>([&](auto cc) {
            constexpr int c = decltype(cc)::value;
            V x;
            if constexpr (G::E == 4) { x.x = v[4 * c]; x.y = v[4 * c + 1]; x.z = v[4 * c + 2]; x.w = v[4 * c + 3]; }
            else { x.x = v[2 * c]; x.y = v[2 * c + 1]; }
            row[c] = x;
        });
    }
    __syncwarp();

    // sum runs of equal targets (lists are sorted by target), one atomicAdd per coefficient and run.  Run heads are found
    // with one ballot; inside a run the row loop has warp-uniform bounds, so its loads are independent and pipeline.
    const T* smT = reinterpret_cast<const T*>(sm);
    T* out = reinterpret_cast<T*>(a.out);
    constexpr int RS = G::KSB * G::E;  // shared row stride in elements
    const int prev = __shfl_up_sync(0xffffffffu, gt, 1);
    unsigned heads = __ballot_sync(0xffffffffu, lane == 0 || gt != prev);
    while (heads) {
        const int r0 = __ffs(heads) - 1;
        heads &= heads - 1;
        const int r1 = heads ? __ffs(heads) - 1 : 32;
        const int t = __shfl_sync(0xffffffffu, gt, r0);
        if (t < 0) continue;  // padding lanes / empty boxes
        T acc[G::NJ];
#pragma unroll
        for (int j = 0; j < G::NJ; ++j) acc[j] = T(0);
#pragma unroll 8
        for (int r = r0; r < r1; ++r) {
#pragma unroll
            for (int j = 0; j < G::NJ; ++j)
                if (lane + 32 * j < G::K) acc[j] += smT[r * RS + lane + 32 * j];
        }
#pragma unroll
        for (int j = 0; j < G::NJ; ++j)
            if (lane + 32 * j < G::K) atomicAdd(out + (int64_t)t * G::Kp + lane + 32 * j, acc[j]);
    }
}

template <typename T, int P, int KIND, int XW = 1, bool GEO = false>
void launch(const XArgs& a, cudaStream_t st) {
    using G = Geo<T, P>;
    constexpr size_t smem = (size_t)XW * 32 * G::KSB * 16 + XW * 8;  // rows + one mbarrier per warp
    static AttrOnce once;
    once.ensure(a.device, [&] { FMM_CUDA_CHECK(cudaFuncSetAttribute(xlate_fast_k<T, P, KIND, XW, GEO>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); });
    const unsigned grid = (unsigned)((a.n + XW * 32 - 1) / (XW * 32));
    xlate_fast_k<T, P, KIND, XW, GEO><<<grid, XW * 32, smem, st>>>(a);
}


// Deterministic M2L (fmm_plan_set_deterministic): ONE WARP PER TARGET BOX walks the box's row of the weak list (CSR by target) in
// batches of 32 pairs and keeps the sums of the translated rows in registers, batch after batch and row after row in list order;
// the single contributor of a row of the local array adds its total at the end.  No floating-point atomics whose order could vary,
// at the price of idle lanes in the last batch of every row (~9 % at config 2) and of the plan-time geometry records (their batches
// are cut differently).
template <typename T, int P, int XW>
__global__ void __launch_bounds__(XW * 32, xlate_warps_per_sm<T, P>() / XW) m2l_row_k(XArgs a) {
    using G = Geo<T, P>;
    using V = typename Vec16<T>::type;
    extern __shared__ __align__(16) unsigned char smraw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    V* sm = reinterpret_cast<V*>(smraw) + (size_t)warp * 32 * G::KSB;
    const int64_t ti = (int64_t)blockIdx.x * XW + warp;
    if (ti >= a.n) return;
    const int gt = (int)(a.first + ti);
    const int64_t e0 = a.woff[gt], e1 = a.woff[gt + 1];
    if (e0 == e1) return;
    constexpr uint32_t ROWB = G::CH * 16;
    const uint32_t bar = smem_u32(reinterpret_cast<unsigned long long*>(smraw + (size_t)XW * 32 * G::KSB * 16) + warp);
    if (lane == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncwarp();
    const T* sc = reinterpret_cast<const T*>(a.scale);
    const T* scs = reinterpret_cast<const T*>(a.scale_s);
    const double tx = a.ctr[3 * (int64_t)gt], ty = a.ctr[3 * (int64_t)gt + 1], tz = a.ctr[3 * (int64_t)gt + 2];
    const T a_new = sc[gt];
    const T* smT = reinterpret_cast<const T*>(sm);
    constexpr int RS = G::KSB * G::E;
    T acc[G::NJ];
#pragma unroll
    for (int j = 0; j < G::NJ; ++j) acc[j] = T(0);
    uint32_t phase = 0;
#pragma unroll 1
    for (int64_t eb = e0; eb < e1; eb += 32) {
        const int64_t e = eb + lane;
        const int gs = e < e1 ? a.src[e] : -1;
        const unsigned vmask = __ballot_sync(0xffffffffu, gs >= 0);
        {
            const int gprev = __shfl_up_sync(0xffffffffu, gs, 1);
            const bool head = lane == 0 || gs < 0 || gprev < 0 || gs != gprev + 1 || G::KSB != G::CH;
            const unsigned hm = __ballot_sync(0xffffffffu, head);
            const unsigned above = lane == 31 ? 0u : (hm >> (lane + 1));
            const int len = above ? __ffs(above) : 32 - lane;
            if (head && gs >= 0)
                bulk_g2s(smem_u32(sm + lane * G::KSB), reinterpret_cast<const char*>(a.in) + (int64_t)gs * ROWB, (uint32_t)len * ROWB, bar);
        }
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)__popc(vmask) * ROWB);
        T bx = T(0), by = T(0), bz = T(1), a_old = T(1);
        if (gs >= 0) {
            bx = (T)(a.ctr_s[3 * (int64_t)gs] - tx);
            by = (T)(a.ctr_s[3 * (int64_t)gs + 1] - ty);
            bz = (T)(a.ctr_s[3 * (int64_t)gs + 2] - tz);
            a_old = scs[gs];
        }
        mbar_wait(bar, phase);
        phase ^= 1u;
        V* row = sm + lane * G::KSB;
        if (gs >= 0) {
            T v[G::KV];
            sfor<G::CH>([&](auto cc) {
                constexpr int c = decltype(cc)::value;
                const V x = row[c];
                if constexpr (G::E == 4) { v[4 * c] = x.x; v[4 * c + 1] = x.y; v[4 * c + 2] = x.z; v[4 * c + 3] = x.w; }
                else { v[2 * c] = x.x; v[2 * c + 1] = x.y; }
            });
            translate_qz<T, P, 1, qz_mode<T>()>(v, bx, by, bz, a_old, a_new);
            sfor<G::CH>([&](auto cc) {
                constexpr int c = decltype(cc)::value;
                V x;
                if constexpr (G::E == 4) { x.x = v[4 * c]; x.y = v[4 * c + 1]; x.z = v[4 * c + 2]; x.w = v[4 * c + 3]; }
                else { x.x = v[2 * c]; x.y = v[2 * c + 1]; }
                row[c] = x;
            });
        }
        __syncwarp();
        const int nv = (int)min((int64_t)32, e1 - eb);
#pragma unroll 4
        for (int r = 0; r < nv; ++r) {
#pragma unroll
            for (int j = 0; j < G::NJ; ++j)
                if (lane + 32 * j < G::K) acc[j] += smT[r * RS + lane + 32 * j];
        }
        __syncwarp();  // every lane has read the rows before the next batch's bulk copies overwrite them
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    T* out = reinterpret_cast<T*>(a.out) + (int64_t)gt * G::Kp;
#pragma unroll
    for (int j = 0; j < G::NJ; ++j)
        if (lane + 32 * j < G::K) out[lane + 32 * j] += acc[j];
}

template <typename T, int P>
void launch_row(const XArgs& a, cudaStream_t st) {
    using G = Geo<T, P>;
    constexpr int XW = 1;  // rows differ in length: one warp per CTA (see xlate_fast_k)
    constexpr size_t smem = (size_t)XW * 32 * G::KSB * 16 + XW * 8;
    static AttrOnce once;
    once.ensure(a.device, [&] { FMM_CUDA_CHECK(cudaFuncSetAttribute(m2l_row_k<T, P, XW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); });
    m2l_row_k<T, P, XW><<<(unsigned)((a.n + XW - 1) / XW), XW * 32, smem, st>>>(a);
}

template <typename T>
bool dispatch_row(int p, const XArgs& a, cudaStream_t st) {
    switch (p) {
#define FMM_CASE(PP) case PP: launch_row<T, PP>(a, st); return true;
        FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
#undef FMM_CASE
        default: return false;
    }
}

template <typename T, int KIND>
bool dispatch(int p, const XArgs& a, cudaStream_t st) {
    switch (p) {
#define FMM_CASE(PP) case PP: \
        if constexpr (sizeof(T) == 4 && KIND == 1) { if (a.geo) { launch<T, PP, KIND, 1, true>(a, st); return true; } } \
        launch<T, PP, KIND, 1, false>(a, st); return true;
        FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
#undef FMM_CASE
#define FMM_CASE(PP) case PP: if constexpr (sizeof(T) == 4) { launch<T, PP, KIND, 1, false>(a, st); return true; } return false;
        FMM_CASE(9) FMM_CASE(10) FMM_CASE(11) FMM_CASE(12)
#undef FMM_CASE
        default: return false;
    }
}

}  // namespace

// plan time (fp32, p <= 8): the geometry record of every weak pair, 1 KB per batch of 32 pairs: ct[32], st[32], cp[32], sp[32],
// 1/r[32], x1[32], x2[32] (float) and the target id[32] (int; -1 for the padding of the last batch) -- what xlate_geometry computes
namespace {
__global__ void m2l_geo_prepare_k(int64_t n, const int32_t* __restrict__ tgt, const int32_t* __restrict__ src, const double* __restrict__ ctr,
                                  const float* __restrict__ scale, const double* __restrict__ ctr_s, const float* __restrict__ scale_s, float* __restrict__ geo) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nb = (n + 31) >> 5;
    if (e >= (nb << 5)) return;
    float ct_ = 1.f, st_ = 0.f, cp_ = 1.f, sp_ = 0.f, rinv = 0.f, x1 = 0.f, x2 = 0.f;
    int gt = -1;
    if (e < n) {
        const int gs = src[e];
        gt = tgt[e];
        const float bx = (float)(ctr_s[3 * (int64_t)gs] - ctr[3 * (int64_t)gt]);
        const float by = (float)(ctr_s[3 * (int64_t)gs + 1] - ctr[3 * (int64_t)gt + 1]);
        const float bz = (float)(ctr_s[3 * (int64_t)gs + 2] - ctr[3 * (int64_t)gt + 2]);
        xr::xlate_geometry<float, 1>(bx, by, bz, scale_s[gs], scale[gt], ct_, st_, cp_, sp_, rinv, x1, x2);
    }
    float* rec = geo + (e >> 5) * 256 + (e & 31);
    rec[0] = ct_; rec[32] = st_; rec[64] = cp_; rec[96] = sp_; rec[128] = rinv; rec[160] = x1; rec[192] = x2;
    reinterpret_cast<int*>(rec)[224] = gt;
}
}  // namespace

bool m2l_geo_wanted(int p, fmm_dtype dt) { return dt == FMM_F32 && p >= 1 && p <= 8; }

// Geometry records of the weak list (28 + 4 bytes per pair; they depend on the positions only, so they are written once per plan).
// The list is cut into the two segments that the evaluate schedule launches separately -- the pairs whose target is above the leaf
// level, [0, w_leaf), and the leaf-level pairs [w_leaf, n_weak) -- each with its own batches of 32.
void m2l_geo_prepare(Plan& P, cudaStream_t st) {
    const int64_t w_leaf = (!P.S && (int64_t)P.weak_level_off.size() > P.L) ? P.weak_level_off[P.L] : 0;
    const int64_t seg_e0[2] = {0, w_leaf}, seg_n[2] = {w_leaf, P.n_weak - w_leaf};
    P.m2l_seg_e0[0] = 0; P.m2l_seg_e0[1] = w_leaf;
    P.m2l_seg_rec[0] = 0; P.m2l_seg_rec[1] = (seg_n[0] + 31) >> 5;
    const int64_t nb = P.m2l_seg_rec[1] + ((seg_n[1] + 31) >> 5);
    P.m2l_geo.alloc((size_t)nb * 256);
    const Plan& PS = P.S ? *P.S : P;
    for (int g = 0; g < 2; ++g) {
        if (seg_n[g] <= 0) continue;
        const int64_t nbg = (seg_n[g] + 31) >> 5;
        m2l_geo_prepare_k<<<(unsigned)((nbg * 32 + 255) / 256), 256, 0, st>>>(seg_n[g], P.weak_tgt.p + seg_e0[g], P.weak_src.p + seg_e0[g], P.box_ctr.p,
                                                                              reinterpret_cast<const float*>(P.box_scale.p), PS.box_ctr.p,
                                                                              reinterpret_cast<const float*>(PS.box_scale.p), P.m2l_geo.p + P.m2l_seg_rec[g] * 256);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
}

// FP32 / FP64 arithmetic instructions of ONE translation as these kernels execute it (operator arithmetic only: the geometry,
// addressing, staging and run sums are not counted) -- the flop count behind bench.py's roofline line.  w = {FMA, MUL, ADD}.
void xlate_work(int p, fmm_dtype dt, int kind, int64_t w[3]) {
    w[0] = w[1] = w[2] = 0;
    if (p < 1 || p > ct::PF) return;
    const int64_t K = (int64_t)(p + 1) * (p + 1), rows = K - 1, nnz = ct::bnnz(p) - 1;  // degree 0 is never touched
    const int64_t zpairs = (int64_t)p * (p + 1) / 2;                                    // (m, -m) pairs of all degrees
    const int n_trig = 4;                                                              // cos / sin tables built per translation (Q Z loop: one per rotation)
    int64_t fma = 0, mul = 0;
    fma += (int64_t)n_trig * p * 2; mul += (int64_t)n_trig * p * 2;                      // addition-theorem recurrences
    fma += 4 * zpairs * 2; mul += 4 * zpairs * 2;                                      // four azimuthal rotations
    fma += 4 * (nnz - rows); mul += 4 * rows;                                          // four applications of Q (or B, B^T)
    if (kind != 2) mul += rows + p;                                                    // source scaling x2^n
    for (int m = -p; m <= p; ++m) {
        const int64_t cnt = p - (m < 0 ? -m : m) + 1;
        if (kind == 1) { mul += cnt; fma += cnt * (cnt - 1); }                         // M2L z-shift: dense cnt x cnt block
        else { fma += cnt * (cnt - 1) / 2; mul += cnt * (cnt - 1) / 2; }               // M2M / L2L: triangular, weight = const * power
    }
    mul += p + (kind == 0 ? 0 : K);                                                    // powers of x1; output scaling (M2L, L2L)
    (void)dt;
    w[0] = fma; w[1] = mul; w[2] = 0;
}

// state vector in registers (this file): p <= 8, and fp32 up to p = 12 (169 + 50 registers of 255, two CTAs of four warps per SM);
// fp64 9 <= p <= 12: state vector in shared memory (xlate_smem.cu)
static bool reg_kernel(int p, fmm_dtype dt) { return p >= 1 && (p <= 8 || (p <= 12 && dt == FMM_F32)); }
bool xlate_fast_available(int p, fmm_dtype dt) { return (dt == FMM_F32 || dt == FMM_F64) && (reg_kernel(p, dt) || xlate_smem_available(p, dt)); }

// deterministic M2L over all target boxes (p <= 8): see m2l_row_k
bool m2l_row_available(int p, fmm_dtype dt) { return (dt == FMM_F32 || dt == FMM_F64) && p >= 1 && p <= 8; }
void m2l_row_launch(const Plan& P, cudaStream_t st) {
    XArgs a{};
    a.device = P.device;
    a.first = 0;
    a.n = P.n_boxes;
    a.woff = P.weak_off.p;
    a.src = P.weak_src.p;
    a.ctr = a.ctr_s = P.box_ctr.p;
    a.scale = a.scale_s = P.box_scale.p;
    a.in = P.Mc.p;
    a.out = P.Lc.p;
    if (P.S) { a.ctr_s = P.S->box_ctr.p; a.scale_s = P.S->box_scale.p; a.in = P.S->Mc.p; }
    if (P.n_weak <= 0) return;
    const bool ok = P.dtype == FMM_F64 ? dispatch_row<double>(P.p, a, st) : dispatch_row<float>(P.p, a, st);
    if (!ok) { set_error("no deterministic register M2L kernel for this order"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
}

void xlate_fast_launch(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    if (!reg_kernel(P.p, P.dtype)) { xlate_smem_launch(P, kind, level, st, e0, e1); return; }
    XArgs a{};
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
        if (P.S) { a.ctr_s = P.S->box_ctr.p; a.scale_s = P.S->box_scale.p; a.in = P.S->Mc.p; }  // sources in their own hierarchy
        // geometry records: usable when [e0, e1) starts at a segment start and does not straddle the two segments
        if (P.m2l_geo.p) {
            const int64_t w = P.m2l_seg_e0[1];
            if (e0 == 0 && (e1 <= w || w == 0)) a.geo = P.m2l_geo.p + P.m2l_seg_rec[w == 0 ? 1 : 0] * 256;
            else if (e0 == w) a.geo = P.m2l_geo.p + P.m2l_seg_rec[1] * 256;
            else if (e0 == 0 && e1 > w) {  // both segments: two launches
                xlate_fast_launch(P, 1, level, st, 0, w);
                xlate_fast_launch(P, 1, level, st, w, e1);
                return;
            }
        }
    } else {
        const int64_t nch = (int64_t)1 << (P.s * level);  // children on `level`
        a.first = e1 < 0 ? 0 : e0;
        a.n = e1 < 0 ? nch : e1 - e0;
        a.off_parent = P.level_off[level - 1];
        a.off_child = P.level_off[level];
        a.in = kind == 0 ? P.Mc.p : P.Lc.p;
        a.out = kind == 0 ? P.Mc.p : P.Lc.p;
    }
    if (a.n <= 0) return;
    bool ok = false;
    if (P.dtype == FMM_F64) {
        if (kind == 0) ok = dispatch<double, 0>(P.p, a, st);
        else if (kind == 1) ok = dispatch<double, 1>(P.p, a, st);
        else ok = dispatch<double, 2>(P.p, a, st);
    } else if (kind == 0) ok = dispatch<float, 0>(P.p, a, st);
    else if (kind == 1) ok = dispatch<float, 1>(P.p, a, st);
    else ok = dispatch<float, 2>(P.p, a, st);
    if (!ok) { set_error("no register translation kernel for this order"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }
}

}  // namespace fmm
