// xlate_fast.cu -- register ("fast") translation kernels: M2M (a5), M2L (a6) and L2L (a7) with ONE THREAD PER TRANSLATION.
//
// The operator is the paper's rotate / shift-along-z / rotate-back (App. B) in the
// normalised, length-scaled representation of tables.cu, where rotations are orthogonal and the polar rotation factors
// as Q(theta) = B Z(theta) B^T with constant matrices B (rot_tables.cuh).  One translation is
//     Z(-phi) B Z(-theta) B^T  [z-shift]  B Z(theta) B^T Z(phi)
// i.e. four azimuthal rotations (2 FP32 instructions per coefficient), four applications of the constant, 3/4-empty B
// (247 MACs each at p=8) and one O(p^3) z-shift (489 MACs at p=8): about 2.3 k FP32 instructions at p=8.
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
// MODE 0 1.66 ms (255 registers either way; MODE 0 spills a little more).
template <typename T> constexpr int qz_mode() { return sizeof(T) == 4 ? 0 : 2; }

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
};

// XW warps per CTA; SYNC = lockstep barriers (all warps then run the operator, also on padding lanes)
template <typename T, int P, int KIND, int XW, bool SYNC>
__global__ void __launch_bounds__(XW * 32, sizeof(T) == 8 ? 1 : (XW == 8 ? 2 : (XW == 4 ? 4 : 1))) xlate_fast_k(XArgs a) {
    using G = Geo<T, P>;
    using V = typename Vec16<T>::type;
    extern __shared__ __align__(16) unsigned char smraw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    V* sm = reinterpret_cast<V*>(smraw) + (size_t)warp * 32 * G::KSB;
    const int64_t e = ((int64_t)blockIdx.x * XW + warp) * 32 + lane;
    int gs = -1, gt = -1;
    if (e < a.n) {
        if constexpr (KIND == 1) { gs = a.src[e]; gt = a.tgt[e]; }
        else {
            const int64_t gc = a.off_child + e, gp = a.off_parent + (e >> a.s);
            if (a.box_count[gc] > 0) {
                if constexpr (KIND == 0) { gs = (int)gc; gt = (int)gp; }
                else { gs = (int)gp; gt = (int)gc; }
            }
        }
    }
    const unsigned vmask = __ballot_sync(0xffffffffu, gs >= 0);
    if constexpr (!SYNC) {
        if (vmask == 0) return;
    }

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
    if (gs >= 0) {
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
    if (SYNC || gs >= 0) {
        sfor<G::CH>([&](auto cc) {
            constexpr int c = decltype(cc)::value;
            const V x = row[c];
            if constexpr (G::E == 4) { v[4 * c] = x.x; v[4 * c + 1] = x.y; v[4 * c + 2] = x.z; v[4 * c + 3] = x.w; }
            else { v[2 * c] = x.x; v[2 * c + 1] = x.y; }
        });
        translate_qz<T, P, KIND, qz_mode<T>()>(v, bx, by, bz, a_old, a_new);
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

template <typename T, int P, int KIND, int XW = 4, bool SYNC = false>
void launch(const XArgs& a, cudaStream_t st) {
    using G = Geo<T, P>;
    constexpr size_t smem = (size_t)XW * 32 * G::KSB * 16 + XW * 8;  // rows + one mbarrier per warp
    static AttrOnce once;
    once.ensure(a.device, [&] { FMM_CUDA_CHECK(cudaFuncSetAttribute(xlate_fast_k<T, P, KIND, XW, SYNC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); });
    const unsigned grid = (unsigned)((a.n + XW * 32 - 1) / (XW * 32));
    xlate_fast_k<T, P, KIND, XW, SYNC><<<grid, XW * 32, smem, st>>>(a);
}

// fp64 M2L at p >= 7 (255 registers, 2 warps per scheduler): the warps of a CTA walk the code in lockstep (SYNC), which shares
// instruction-cache lines: p = 8 2.48 -> 2.01 ms on B200; at p <= 6 and in fp32 (4 warps per scheduler) lockstep costs more than it saves.
template <typename T, int KIND>
bool dispatch(int p, const XArgs& a, cudaStream_t st) {
    switch (p) {
#define FMM_CASE(PP) case PP: launch<T, PP, KIND, 4, false>(a, st); return true;
        FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
#undef FMM_CASE
        default: return false;
    }
}

}  // namespace

// p <= 8: state vector in registers (this file); 9 <= p <= 12: state vector in shared memory (xlate_smem.cu)
bool xlate_fast_available(int p, fmm_dtype dt) { return (dt == FMM_F32 || dt == FMM_F64) && ((p >= 1 && p <= 8) || xlate_smem_available(p, dt)); }

void xlate_fast_launch(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1) {
    if (P.p > 8) { xlate_smem_launch(P, kind, level, st, e0, e1); return; }
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
    } else {
        a.n = (int64_t)1 << (P.s * level);  // children on `level`
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
