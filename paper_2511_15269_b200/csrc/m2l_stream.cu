// m2l_stream.cu -- fp32 M2L (a6), one weak pair per thread like xlate_fast.cu KIND 1, but software-pipelined:
//
//   * the plan stores the weak list a second time in BATCHES of 32 pairs that never straddle two targets (`wpad_src`,
//     padded with -1; `wpad_tgt` one target id per batch; plan.cu build_m2l_batches).  About 10 % of the lanes are padding
//     at config 2 (172 sources per target), which buys three things:
//   * a warp works through NB consecutive batches and, while it computes batch i, the source rows of batch i+1 are already
//     on their way into its (single) shared-memory buffer by TMA bulk copies, the box geometry of batch i+1 by cp.async,
//     and the source ids of batch i+2 into registers -- the load latency that took a third of a warp's life in the
//     one-batch-per-warp kernel is paid once per NB batches;
//   * all 32 results of a batch belong to one target, so they are summed by a recursive-halving reduce-scatter in registers
//     (shuffles only, no staging buffer -- which is what leaves room for the prefetch buffer) and added to D with three
//     coalesced atomicAdd per lane.
//
// Operator and numerics are those of translate_reg<float, P, 1> (xlate_reg.cuh / xlate_fast.cu): App. B.
#include "tma.cuh"
#include "xlate_reg.cuh"

namespace fmm {

namespace {

using namespace xr;

constexpr int NB = 8;   // consecutive batches per warp

template <int P>
struct SGeo {
    static constexpr int K = (P + 1) * (P + 1);
    static constexpr int Kp = (K + 3) & ~3;
    static constexpr int CH = Kp / 4;                   // 16-byte chunks per row
    static constexpr int KSB = (CH & 1) ? CH : CH + 1;  // shared row stride in 16-byte units (odd)
    static constexpr int KV = CH * 4;
    static constexpr int NJ = (KV + 31) / 32;           // results per lane after the reduce-scatter
    static constexpr int KP = NJ * 32;
    static constexpr size_t ROWS = (size_t)32 * KSB * 16;
    static constexpr size_t SMEM_WARP = ROWS + 32 * 6 * sizeof(double) + 32 * 2 * sizeof(float) + 16;
};

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// sum over the 32 lanes of v[0..KV) (entries >= KV count as zero): afterwards lane l holds the sums of coefficients
// NJ*l .. NJ*l + NJ-1 in out[].  KP/2 + KP/4 + ... + NJ shuffles.
template <int KV, int KP, int NJ>
__device__ __forceinline__ void reduce_scatter(const float (&v)[KV], float (&out)[NJ], int lane) {
    constexpr int H = KP / 2;
    float w[H];
    {
        const bool up = (lane & 16) != 0;
        sfor<H>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const float lo = i < KV ? v[i < KV ? i : 0] : 0.f;
            const float hi = i + H < KV ? v[i + H < KV ? i + H : 0] : 0.f;
            const float send = up ? lo : hi, keep = up ? hi : lo;
            w[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        });
    }
#pragma unroll
    for (int bit = 8, h = H / 2; bit > 0; bit >>= 1, h >>= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const float send = up ? w[i] : w[i + h], keep = up ? w[i + h] : w[i];
            w[i] = keep + __shfl_xor_sync(0xffffffffu, send, bit);
        }
    }
#pragma unroll
    for (int j = 0; j < NJ; ++j) out[j] = w[j];
}

// SW warps per CTA.  SYNC: the warps of the CTA run the operator in barrier lockstep (they then fetch the same instruction
// lines at the same time); every warp executes NB iterations, idle ones on zero vectors.
template <int P, int SW, bool SYNC>
__global__ void __launch_bounds__(SW * 32, 16 / SW)
m2l_stream_k(int64_t b_begin, int64_t b_end, const int32_t* __restrict__ wpad_src, const int32_t* __restrict__ wpad_tgt,
             const double* __restrict__ ctr, const float* __restrict__ scale, const float* __restrict__ Mc, float* __restrict__ Lc) {
    using G = SGeo<P>;
    extern __shared__ __align__(16) unsigned char smraw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* wbase = smraw + (size_t)warp * G::SMEM_WARP;
    float4* rows = reinterpret_cast<float4*>(wbase);
    double* gsm = reinterpret_cast<double*>(wbase + G::ROWS);                       // [6][32]: source centre, target centre
    float* ssm = reinterpret_cast<float*>(wbase + G::ROWS + 32 * 6 * sizeof(double));  // [2][32]: a_source, a_target
    const uint32_t bar = smem_u32(wbase + G::ROWS + 32 * 6 * sizeof(double) + 32 * 2 * sizeof(float));
    int64_t b = b_begin + ((int64_t)blockIdx.x * SW + warp) * NB;
    const int64_t bend = b + NB < b_end ? b + NB : b_end;
    if constexpr (!SYNC) {
        if (b >= bend) return;
    }
    if (lane == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncwarp();

    constexpr uint32_t ROWB = G::CH * 16;
    // start the copies of one batch: rows by TMA (one bulk copy per run of consecutive source ids), geometry by cp.async
    auto issue = [&](int gs, int gt) {
        const int gprev = __shfl_up_sync(0xffffffffu, gs, 1);
        const bool head = lane == 0 || gs < 0 || gprev < 0 || gs != gprev + 1 || G::KSB != G::CH;
        const unsigned hm = __ballot_sync(0xffffffffu, head);
        const unsigned vm = __ballot_sync(0xffffffffu, gs >= 0);
        const unsigned above = lane == 31 ? 0u : (hm >> (lane + 1));
        const int len = above ? __ffs(above) : 32 - lane;
        if (head && gs >= 0)
            bulk_g2s(smem_u32(rows + lane * G::KSB), reinterpret_cast<const char*>(Mc) + (int64_t)gs * ROWB, (uint32_t)len * ROWB, bar);
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)__popc(vm) * ROWB);
        if (gs >= 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                cp_async8(gsm + k * 32 + lane, ctr + 3 * (int64_t)gs + k);
                cp_async8(gsm + (3 + k) * 32 + lane, ctr + 3 * (int64_t)gt + k);
            }
            cp_async4(ssm + lane, scale + gs);
            cp_async4(ssm + 32 + lane, scale + gt);
        }
    };

    int gs = -1, gt = -1;
    if (b < bend) {
        gs = wpad_src[b * 32 + lane];
        gt = wpad_tgt[b];
        issue(gs, gt);
    }
    int gs_n = -1, gt_n = -1;
    if (b + 1 < bend) { gs_n = wpad_src[(b + 1) * 32 + lane]; gt_n = wpad_tgt[b + 1]; }

    for (int it = 0; SYNC ? it < NB : b < bend; ++b, ++it) {
        const bool active = b < bend;
        if (active) {
            mbar_wait(bar, it & 1);
            cp_async_wait_all();
        } else gs = -1;
        __syncwarp();
        float v[G::KV];
        float bx = 0.f, by = 0.f, bz = 1.f, a_old = 1.f, a_new = 1.f;
        {
            const float4* row = rows + lane * G::KSB;
            sfor<G::CH>([&](auto cc) {
                constexpr int c = decltype(cc)::value;
                const float4 x = gs >= 0 ? row[c] : make_float4(0.f, 0.f, 0.f, 0.f);  // padding lanes translate a zero vector
                v[4 * c] = x.x; v[4 * c + 1] = x.y; v[4 * c + 2] = x.z; v[4 * c + 3] = x.w;
            });
            if (gs >= 0) {
                bx = (float)(gsm[lane] - gsm[3 * 32 + lane]);
                by = (float)(gsm[32 + lane] - gsm[4 * 32 + lane]);
                bz = (float)(gsm[2 * 32 + lane] - gsm[5 * 32 + lane]);
                a_old = ssm[lane];
                a_new = ssm[32 + lane];
            }
        }
        const int tgt = gt;
        __syncwarp();          // every lane has its row and geometry in registers: the buffers may be refilled
        fence_proxy_async();   // order the generic-proxy reads above before the async-proxy writes below
        if (b + 1 < bend) {
            gs = gs_n; gt = gt_n;
            issue(gs, gt);
            if (b + 2 < bend) { gs_n = wpad_src[(b + 2) * 32 + lane]; gt_n = wpad_tgt[b + 2]; }
        }

        translate_reg<float, P, 1, SYNC>(v, bx, by, bz, a_old, a_new);

        float out[G::NJ];
        reduce_scatter<G::KV, G::KP, G::NJ>(v, out, lane);
#pragma unroll
        for (int j = 0; j < G::NJ; ++j)
            if (active && G::NJ * lane + j < G::K) atomicAdd(Lc + (int64_t)tgt * G::Kp + G::NJ * lane + j, out[j]);
    }
}

template <int P, int SW = 4, bool SYNC = false>
void launch_stream(const Plan& Pl, cudaStream_t st, int64_t b0, int64_t b1) {
    using G = SGeo<P>;
    constexpr size_t smem = (size_t)SW * G::SMEM_WARP;
    static bool attr_set = false;
    if (!attr_set) {
        FMM_CUDA_CHECK(cudaFuncSetAttribute(m2l_stream_k<P, SW, SYNC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    const int64_t per_cta = (int64_t)SW * NB;
    const unsigned grid = (unsigned)((b1 - b0 + per_cta - 1) / per_cta);
    m2l_stream_k<P, SW, SYNC><<<grid, SW * 32, smem, st>>>(b0, b1, Pl.wpad_src.p, Pl.wpad_tgt.p, Pl.box_ctr.p, (const float*)Pl.box_scale.p,
                                                 (const float*)Pl.Mc.p, (float*)Pl.Lc.p);
}

}  // namespace

bool m2l_stream_available(int p, fmm_dtype dt) { return dt == FMM_F32 && p >= 1 && p <= 8; }

// batches [b0, b1) of the padded weak list (plan.cu build_m2l_batches); results are ADDED to Lc
void m2l_stream_launch(const Plan& P, cudaStream_t st, int64_t b0, int64_t b1) {
    if (b1 <= b0) return;
    switch (P.p) {
#define FMM_CASE(PP) case PP: launch_stream<PP>(P, st, b0, b1); break;
        FMM_CASE(1) FMM_CASE(2) FMM_CASE(3) FMM_CASE(4) FMM_CASE(5) FMM_CASE(6) FMM_CASE(7) FMM_CASE(8)
#undef FMM_CASE
        default: set_error("no streaming M2L kernel for this order"); throw CudaFail{FMM_ERR_UNSUPPORTED};
    }
}

}  // namespace fmm
