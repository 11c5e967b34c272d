// p2p_fast.cu -- fp32 near field (a9): direct sum over the strong leaf pairs (stage "evdir" PAPER.md:251;
// DESIGN.md reading S3).  Writes (phi_near, grad phi_near) per particle in tree order; the L2P kernel (evaluate.cu) adds the far field,
// scales and scatters to input order (a10).  The kernel depends only on the permuted particles, so run_evaluate launches it
// on a second stream, concurrently with the whole far-field chain.
//
// Mapping (differs from north_star's "one target leaf per CTA": one target leaf per WARP):
//   * a warp owns one target leaf (or a chunk of 32*TPT targets of a large leaf); lanes form ntgp target groups x nsl
//     source slices, every lane keeps TPT targets in registers;
//   * sources are read from `srcg`, a per-evaluate copy of the particles in groups of four, (-x[4], -y[4], -z[4], q[4]) =
//     64 bytes, every leaf padded to whole groups with zero charges (written by the permute kernel).  A warp copies the
//     groups of its source leaves into its private, double-buffered shared-memory tiles with TMA bulk copies
//     (cp.async.bulk + mbarrier: one copy per source leaf, issued by 32 lanes at once), so staging costs a handful of
//     instructions per tile and overlaps with the arithmetic on the previous tile; one LDS.128 per component then brings
//     FOUR sources as two packed pairs;
//   * all FP32 arithmetic of a (target, source-pair) runs as packed f32x2 instructions (FADD2 / FMUL2 / FFMA2, new on
//     sm_100): 13 packed instructions + 2 MUFU.RSQ + 2 (FSETP+FSEL) per two particle pairs.  The FMA pipe issues a packed
//     instruction every other cycle, which leaves the issue slots in between for MUFU, the mask, LDS and the loop;
//   * slices are combined with warp shuffles (no block-level synchronisation anywhere in the kernel).
#include <type_traits>

#include "internal.cuh"
#include "tma.cuh"

namespace fmm {
namespace {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pk(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ float rsq(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// PW = warps per CTA (independent of one another).  One: a CTA's resources are held until its slowest warp is done and the items differ (a leaf has
// 8-27 strong-list entries); measured on B200, P2P of config 2: 4 warps 0.480 ms, 2: 0.477, 1: 0.463 ms; config 4: 0.451 -> 0.405 ms.  Leaves of
// more than 128 particles keep four warps per CTA: their items are long, and neighbours on one SM share the staged sources' L2 lines
// (N = 1e7, leaves of 488: 38.8 against 42.5 ms).
constexpr int TG = 64;  // groups (of four sources, 64 bytes) per warp tile; two tiles per warp = 8 KB of shared memory

// Source particles come from `srcg`: per leaf a block of G groups; group = 16 floats (-x[4], -y[4], -z[4], q[4]); slots beyond
// the leaf population hold zeros (zero charge), so whole groups can be used without masks.
// WF = false: potential only (fmm_evaluate with d_field == NULL): 7 instead of 13 packed instructions per two pairs
// ZT = true: tiles without a touching leaf pair skip the zero-distance mask (pays for leaves of >~ 32 particles; with small
// leaves every tile holds the target leaf itself)
template <int TPT, int HS, bool WF, bool ZT, int PW = 1>
__global__ void __launch_bounds__(PW * 32) p2p_fast_k(const float4* __restrict__ pq, const float* __restrict__ srcg, int G,
                                                      const int32_t* __restrict__ leaf_start, const int32_t* __restrict__ leaf_cnt,
                                                      const P2PItem* __restrict__ items, const int32_t* __restrict__ strong_src,
                                                      const uint8_t* __restrict__ strong_touch, float4* __restrict__ near, int64_t n_items, int nchunk) {
    __shared__ __align__(128) float sm[PW][2][TG * 16];
    __shared__ __align__(8) unsigned long long bars[PW][2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t item = (int64_t)blockIdx.x * PW + warp;
    if (item >= n_items) return;
    const int64_t iw = item / nchunk;
    const int chunk = (int)(item - iw * nchunk);
    const P2PItem wi = items[iw];  // one segment of the strong list of one target leaf
    const bool multi = wi.e1 < 0;
    const int tst = wi.start, tcnt = wi.cnt;
    const int t0 = chunk * 32 * TPT;
    if (t0 >= tcnt) return;
    const int tn = min(tcnt - t0, 32 * TPT);
    const int ntg = (tn + TPT - 1) / TPT;
    int lg = 0;
    while ((1 << lg) < ntg) ++lg;
    const int ntgp = 1 << lg, nsl = 32 >> lg;
    const int tg = lane & (ntgp - 1), sl = lane >> lg;

    const uint32_t bar0 = smem_u32(&bars[warp][0]), buf0 = smem_u32(&sm[warp][0][0]);
    if (lane == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    // targets of this lane (the compiler turns pk(v, v) into a broadcast operand of the packed instructions)
    u64 TX[TPT], TY[TPT], TZ[TPT], PH[TPT], GX[TPT], GY[TPT], GZ[TPT];
#pragma unroll
    for (int k = 0; k < TPT; ++k) {
        const int ti = tg * TPT + k;
        float4 v = make_float4(1e18f, 1e18f, 1e18f, 0.f);  // unused slots are parked far away; their sums are discarded
        if (ti < tn) v = pq[tst + t0 + ti];
        TX[k] = pk(v.x, v.x);
        TY[k] = pk(v.y, v.y);
        TZ[k] = pk(v.z, v.z);
        PH[k] = GX[k] = GY[k] = GZ[k] = 0ull;
    }

    int64_t e = wi.e0;
    const int64_t e1 = multi ? ~wi.e1 : wi.e1;
    int sub = 0;  // groups of entry e already consumed

    // producer: fill tile `b` with up to TG groups starting at the cursor (e, sub); every lane issues the bulk copy of "its" entry
    // zf: set if an entry copied into the tile may hold a source at zero distance from a target (strong_touch): only such
    // tiles run the masked loop (reading S3); pad slots are parked far away by the plan and never coincide with anything
    auto produce = [&](int b, bool& zf) -> int {
        int fill = 0;
        uint32_t bytes = 0;
        zf = false;
        const uint32_t bar = bar0 + 8 * b, buf = buf0 + (uint32_t)b * (TG * 64);
        while (e < e1 && fill < TG) {
            const int nb = (int)min((int64_t)32, e1 - e);
            int c = 0;
            int64_t g0 = 0;
            if (lane < nb) {
                const int ent = strong_src[e + lane];
                g0 = (int64_t)ent * G;
                c = (leaf_cnt[ent] + 3) >> 2;
            }
            if (lane == 0) { g0 += sub; c -= sub; }
            int incl = c;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            const int excl = incl - c;
            const int room = TG - fill;
            const int ni = min(c, room - excl);
            if (ni > 0) {
                bulk_g2s(buf + (uint32_t)(fill + excl) * 64u, srcg + g0 * 16, (uint32_t)ni * 64u, bar);
                bytes += (uint32_t)ni * 64u;
            }
            if constexpr (ZT) zf |= __any_sync(0xffffffffu, ni > 0 && strong_touch[e + lane] != 0);
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            if (total <= room) {
                fill += total;
                e += nb;
                sub = 0;
            } else {
                const unsigned m = __ballot_sync(0xffffffffu, incl > room);
                const int idx = __ffs(m) - 1;
                const int ex = __shfl_sync(0xffffffffu, excl, idx);
                sub = (idx == 0 ? sub : 0) + (room - ex);
                e += idx;
                fill = TG;
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, d);
        if (lane == 0) mbar_expect_tx(bar, bytes);
        return fill;
    };

    bool zf_next = false;
    int ng_next = (e < e1) ? produce(0, zf_next) : 0;
    for (int t = 0; ng_next > 0; ++t) {
        const int b = t & 1;
        const int ng = ng_next;
        const bool zf = zf_next;
        __syncwarp();  // every lane has finished reading the other buffer (tile t-1)
        ng_next = (e < e1) ? produce(b ^ 1, zf_next) : 0;
        mbar_wait(bar0 + 8 * b, (t >> 1) & 1);
        const ulonglong2* T2 = reinterpret_cast<const ulonglong2*>(&sm[warp][b][0]);
        auto run_tile = [&](auto mkc) {
        constexpr bool MK = decltype(mkc)::value;
        for (int j = sl; j < ng; j += nsl) {
            const ulonglong2 xs = T2[4 * j], ys = T2[4 * j + 1], zs = T2[4 * j + 2], qs = T2[4 * j + 3];
            // staged over the NC = HS * TPT independent chains (all distances, then all rsqrt, then the accumulation) so that
            // the MUFU latency of one chain is covered by the arithmetic of the others inside one warp
            constexpr int NC = HS * TPT;
#pragma unroll
            for (int h0 = 0; h0 < 2; h0 += HS) {
                u64 dx[NC], dy[NC], dz[NC], r2[NC];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const int h = h0 + c / TPT, k = c % TPT;
                    const u64 sx = h ? xs.y : xs.x, sy = h ? ys.y : ys.x, sz = h ? zs.y : zs.x;
                    dx[c] = add2(TX[k], sx); dy[c] = add2(TY[k], sy); dz[c] = add2(TZ[k], sz);
                    r2[c] = mul2(dx[c], dx[c]);
                }
#pragma unroll
                for (int c = 0; c < NC; ++c) r2[c] = fma2(dy[c], dy[c], r2[c]);
#pragma unroll
                for (int c = 0; c < NC; ++c) r2[c] = fma2(dz[c], dz[c], r2[c]);
                float ia[NC], ib[NC];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    float a, b2;
                    upk(r2[c], a, b2);
                    ia[c] = rsq(a); ib[c] = rsq(b2);
                }
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const int h = h0 + c / TPT, k = c % TPT;
                    const u64 sq = h ? qs.y : qs.x;
                    float a, b2;
                    upk(r2[c], a, b2);
                    // reading S3: coincident pairs contribute nothing (r^2 below FLT_MIN counts as coincident in fp32)
                    const float ja = (!MK || a >= 1.17549435e-38f) ? ia[c] : 0.f;
                    const float jb = (!MK || b2 >= 1.17549435e-38f) ? ib[c] : 0.f;
                    const u64 inv = pk(ja, jb);
                    if constexpr (WF) {
                        const u64 qi = mul2(sq, inv), inv2 = mul2(inv, inv);
                        const u64 q3 = mul2(qi, inv2);
                        PH[k] = add2(PH[k], qi);
                        GX[k] = fma2(q3, dx[c], GX[k]);
                        GY[k] = fma2(q3, dy[c], GY[k]);
                        GZ[k] = fma2(q3, dz[c], GZ[k]);
                    } else {
                        PH[k] = fma2(sq, inv, PH[k]);
                    }
                }
            }
        }
        };
        if (!ZT || zf) run_tile(std::true_type{});
        else run_tile(std::false_type{});
    }

    // combine the two packed halves, then the source slices (lanes that differ in the bits above lg)
    float ph[TPT], gx[TPT], gy[TPT], gz[TPT];
#pragma unroll
    for (int k = 0; k < TPT; ++k) {
        float a, b;
        upk(PH[k], a, b); ph[k] = a + b;
        upk(GX[k], a, b); gx[k] = a + b;
        upk(GY[k], a, b); gy[k] = a + b;
        upk(GZ[k], a, b); gz[k] = a + b;
    }
    for (int d = ntgp; d < 32; d <<= 1) {
#pragma unroll
        for (int k = 0; k < TPT; ++k) {
            ph[k] += __shfl_xor_sync(0xffffffffu, ph[k], d);
            if constexpr (WF) {
                gx[k] += __shfl_xor_sync(0xffffffffu, gx[k], d);
                gy[k] += __shfl_xor_sync(0xffffffffu, gy[k], d);
                gz[k] += __shfl_xor_sync(0xffffffffu, gz[k], d);
            }
        }
    }
    // every lane now holds the full sums of its group; slice sl writes the targets k with k mod nsl == sl
#pragma unroll
    for (int k = 0; k < TPT; ++k) {
        const int ti = tg * TPT + k;
        // G accumulates +q d / r^3 = -grad phi_near; stored: (phi_near, grad phi_near) in tree order for the L2P finalize
        if ((k & (nsl - 1)) == sl && ti < tn) {
            if (!multi) near[tst + t0 + ti] = make_float4(ph[k], -gx[k], -gy[k], -gz[k]);
            else {  // several segments per leaf: `near` was zeroed by run_evaluate
                float* o = reinterpret_cast<float*>(near + tst + t0 + ti);
                atomicAdd(o, ph[k]);
                if constexpr (WF) { atomicAdd(o + 1, -gx[k]); atomicAdd(o + 2, -gy[k]); atomicAdd(o + 3, -gz[k]); }
            }
        }
    }
}

// 1/sqrt(x) for normal, finite x > 0 (squared distances): the hardware seed (MUFU.RSQ64H, relative error ~2^-22) refined by one
// third-order step  y = y0 + y0 e (1/2 + 3/8 e),  e = 1 - x y0^2  (error ~ (5/16) e^3 < 2^-66): 5 DFMA-class instructions instead
// of the library rsqrt's range checks and two Newton steps.  x = 0 gives NaN, which the caller selects away.
__device__ __forceinline__ double drsqrt(double x) {
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    const double t = x * y0;
    const double e = fma(-t, y0, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(y0 * e, p, y0);
}

// ---- fp64 near field: the same mapping (one target leaf, or one segment of its strong list, per warp; lanes = target groups x
// source slices; TPT targets per lane in registers), plain scalar DFMA arithmetic.  The FP64 pipe runs at half the FP32 rate and
// one (target, source) pair costs ~13 DFMA-class instructions plus a double-precision rsqrt (MUFU.RSQ64H + Newton steps), so a
// source (one 32-byte (x, y, z, q) record) is simply read from `pq` through L1 -- eight lanes of a slice read the same address --
// and no shared-memory staging is needed: 2 loads against ~90 FP64 instructions per source and lane.
// PW64 warps per CTA: this kernel leans on L1 / L2 for its sources, and neighbouring work items (neighbouring leaves) read the same ones.
// One warp per CTA (see p2p_fast_k) wins while the particles fit the L2 and leaves are small (N = 1M, leaves of 30: 1.43 -> 1.39 ms); four warps
// keep neighbours on one SM and win otherwise (N = 1e7, leaves of 19: 5.36 against 5.66 ms; leaves of 256 at N = 2^20: 79 against 90 ms).
template <int TPT, bool WF, int PW64>
__global__ void __launch_bounds__(PW64 * 32, PW64 == 4 ? 4 : 1) p2p_warp64_k(const double4* __restrict__ pq, const double4* __restrict__ pq_s,
                                                        const int32_t* __restrict__ sleaf_start, const int32_t* __restrict__ sleaf_cnt,
                                                        const P2PItem* __restrict__ items, const int32_t* __restrict__ strong_src,
                                                        double4* __restrict__ near, int64_t n_items, int nchunk) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t item = (int64_t)blockIdx.x * PW64 + warp;
    if (item >= n_items) return;
    const int64_t iw = item / nchunk;
    const int chunk = (int)(item - iw * nchunk);
    const P2PItem wi = items[iw];
    const bool multi = wi.e1 < 0;
    const int tst = wi.start, tcnt = wi.cnt;
    const int t0 = chunk * 32 * TPT;
    if (t0 >= tcnt) return;
    const int tn = min(tcnt - t0, 32 * TPT);
    const int ntg = (tn + TPT - 1) / TPT;
    int lg = 0;
    while ((1 << lg) < ntg) ++lg;
    const int ntgp = 1 << lg, nsl = 32 >> lg;
    const int tg = lane & (ntgp - 1), sl = lane >> lg;
    double tx[TPT], ty[TPT], tz[TPT], ph[TPT], gx[TPT], gy[TPT], gz[TPT];
#pragma unroll
    for (int k = 0; k < TPT; ++k) {
        const int ti = tg * TPT + k;
        double4 v = make_double4(1e150, 1e150, 1e150, 0.0);  // unused slots are parked far away; their sums are discarded
        if (ti < tn) v = pq[tst + t0 + ti];
        tx[k] = v.x; ty[k] = v.y; tz[k] = v.z;
        ph[k] = gx[k] = gy[k] = gz[k] = 0.0;
    }
    const int64_t e1 = multi ? ~wi.e1 : wi.e1;
    for (int64_t e = wi.e0; e < e1; ++e) {
        const int sleaf = strong_src[e];
        const int sst = sleaf_start[sleaf], sc = sleaf_cnt[sleaf];
#pragma unroll 2
        for (int j = sl; j < sc; j += nsl) {
            const double4 sv = pq_s[sst + j];
#pragma unroll
            for (int k = 0; k < TPT; ++k) {
                const double dx = tx[k] - sv.x, dy = ty[k] - sv.y, dz = tz[k] - sv.z;
                const double r2 = dx * dx + dy * dy + dz * dz;
                double inv = drsqrt(r2);
                inv = (r2 > 0.0) ? inv : 0.0;  // reading S3: self / coincident pairs contribute nothing (selects away the NaN of r2 = 0)
                const double qi = sv.w * inv;
                ph[k] += qi;
                if constexpr (WF) {
                    const double q3 = qi * (inv * inv);
                    gx[k] -= q3 * dx; gy[k] -= q3 * dy; gz[k] -= q3 * dz;
                }
            }
        }
    }
    for (int d = ntgp; d < 32; d <<= 1) {
#pragma unroll
        for (int k = 0; k < TPT; ++k) {
            ph[k] += __shfl_xor_sync(0xffffffffu, ph[k], d);
            if constexpr (WF) {
                gx[k] += __shfl_xor_sync(0xffffffffu, gx[k], d);
                gy[k] += __shfl_xor_sync(0xffffffffu, gy[k], d);
                gz[k] += __shfl_xor_sync(0xffffffffu, gz[k], d);
            }
        }
    }
#pragma unroll
    for (int k = 0; k < TPT; ++k) {
        const int ti = tg * TPT + k;
        if ((k & (nsl - 1)) == sl && ti < tn) {  // (phi_near, grad phi_near) in tree order for the L2P finalize
            if (!multi) near[tst + t0 + ti] = make_double4(ph[k], gx[k], gy[k], gz[k]);
            else {
                double* o = reinterpret_cast<double*>(near + tst + t0 + ti);
                atomicAdd(o, ph[k]);
                if constexpr (WF) { atomicAdd(o + 1, gx[k]); atomicAdd(o + 2, gy[k]); atomicAdd(o + 3, gz[k]); }
            }
        }
    }
}

}  // namespace

template <int TPT, int HS>
static void p2p_launch_t(const Plan& P, cudaStream_t st, bool wf, int64_t item0, int64_t item1) {
    const int64_t leaf0 = P.level_off[P.L];
    const int nchunk = (P.max_leaf + 32 * TPT - 1) / (32 * TPT);
    if (item1 < 0) { item0 = 0; item1 = P.n_p2p_items; }
    const int64_t n_items = (item1 - item0) * nchunk;
    // separate targets: a target leaf may have an empty strong list and then no work item; its near field must read zero
    if (P.p2p_multi || P.S) FMM_CUDA_CHECK(cudaMemsetAsync(P.near.p, 0, P.near.n, st));
    if (n_items == 0) return;
    const Plan& PS = P.S ? *P.S : P;  // hierarchy of the sources (separate targets)
    auto go = [&](auto pwc) {
        constexpr int PW = decltype(pwc)::value;
        const unsigned grid = (unsigned)((n_items + PW - 1) / PW);
        if (wf) p2p_fast_k<TPT, HS, true, (TPT > 2), PW><<<grid, PW * 32, 0, st>>>((const float4*)P.pq.p, (const float*)PS.srcg.p, PS.src_G, P.box_start.p + leaf0, PS.box_count.p + PS.level_off[PS.L],
                                                  reinterpret_cast<const P2PItem*>(P.p2p_items.p) + item0, P.strong_src.p, P.strong_touch.p, (float4*)P.near.p, n_items, nchunk);
        else p2p_fast_k<TPT, HS, false, (TPT > 2), PW><<<grid, PW * 32, 0, st>>>((const float4*)P.pq.p, (const float*)PS.srcg.p, PS.src_G, P.box_start.p + leaf0, PS.box_count.p + PS.level_off[PS.L],
                                                  reinterpret_cast<const P2PItem*>(P.p2p_items.p) + item0, P.strong_src.p, P.strong_touch.p, (float4*)P.near.p, n_items, nchunk);
    };
    if (P.max_leaf <= 128) go(std::integral_constant<int, 1>{});
    else go(std::integral_constant<int, 4>{});
}

// Targets per lane.  A median-split tree gives every leaf the same population (+-1), so max_leaf decides the lane layout for
// the whole launch: the warp holds ntgp = 8, 16 or 32 target groups of TPT targets (x 4, 2 or 1 source slices); pick the
// layout that wastes the fewest target slots, ties to the fewest groups (most register reuse of a staged source).
// Measured on B200 (P2P stage, CUDA events): config 2 (leaves of 30-31): <TPT, HS> = <4,1> 0.488, <4,2> 0.482, <2,2> 0.525,
// <1,2> 0.494, <8,1> 0.489 ms; config 4 (leaves of 16): <4,*> 0.562, <2,2> 0.433 ms.
static int choose_tpt(int max_leaf) {
    int best = 4;
    double best_eff = -1.0;
    const int m = max_leaf < 1 ? 1 : (max_leaf > 256 ? 256 : max_leaf);  // larger leaves are cut into chunks of 32 * TPT targets
    for (int ntgp = 8; ntgp <= 32; ntgp *= 2) {
        const int tpt = (m + ntgp - 1) / ntgp;
        if (tpt > 8) continue;
        const double eff = (double)m / (tpt * ntgp);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = tpt; }
    }
    return best;
}

void p2p_fast_launch(const Plan& P, cudaStream_t st, bool wf, int64_t i0, int64_t i1) {
    switch (choose_tpt(P.max_leaf)) {
        case 1: p2p_launch_t<1, 2>(P, st, wf, i0, i1); break;
        case 2: p2p_launch_t<2, 2>(P, st, wf, i0, i1); break;
        case 3: p2p_launch_t<3, 2>(P, st, wf, i0, i1); break;
        case 4: p2p_launch_t<4, 2>(P, st, wf, i0, i1); break;
        case 5: p2p_launch_t<5, 1>(P, st, wf, i0, i1); break;
        case 6: p2p_launch_t<6, 1>(P, st, wf, i0, i1); break;
        case 7: p2p_launch_t<7, 1>(P, st, wf, i0, i1); break;
        default: p2p_launch_t<8, 1>(P, st, wf, i0, i1); break;
    }
}

template <int TPT>
static void p2p_launch64_t(const Plan& P, cudaStream_t st, bool wf, int64_t item0, int64_t item1) {
    const Plan& PS = P.S ? *P.S : P;
    const int64_t sleaf0 = PS.level_off[PS.L];
    const int nchunk = (P.max_leaf + 32 * TPT - 1) / (32 * TPT);
    if (item1 < 0) { item0 = 0; item1 = P.n_p2p_items; }
    const int64_t n_items = (item1 - item0) * nchunk;
    if (P.p2p_multi || P.S) FMM_CUDA_CHECK(cudaMemsetAsync(P.near.p, 0, P.near.n, st));
    if (n_items == 0) return;
    auto go = [&](auto pwc) {
        constexpr int PW64 = decltype(pwc)::value;
        const unsigned grid = (unsigned)((n_items + PW64 - 1) / PW64);
        if (wf) p2p_warp64_k<TPT, true, PW64><<<grid, PW64 * 32, 0, st>>>((const double4*)P.pq.p, (const double4*)PS.pq.p, PS.box_start.p + sleaf0, PS.box_count.p + sleaf0,
                                                    reinterpret_cast<const P2PItem*>(P.p2p_items.p) + item0, P.strong_src.p, (double4*)P.near.p, n_items, nchunk);
        else p2p_warp64_k<TPT, false, PW64><<<grid, PW64 * 32, 0, st>>>((const double4*)P.pq.p, (const double4*)PS.pq.p, PS.box_start.p + sleaf0, PS.box_count.p + sleaf0,
                                                    reinterpret_cast<const P2PItem*>(P.p2p_items.p) + item0, P.strong_src.p, (double4*)P.near.p, n_items, nchunk);
    };
    if (PS.N <= 3000000 && P.max_leaf <= 128) go(std::integral_constant<int, 1>{});
    else go(std::integral_constant<int, 4>{});
}

void p2p_fast64_launch(const Plan& P, cudaStream_t st, bool wf, int64_t i0, int64_t i1) {
    switch (choose_tpt(P.max_leaf)) {
        case 1: p2p_launch64_t<1>(P, st, wf, i0, i1); break;
        case 2: p2p_launch64_t<2>(P, st, wf, i0, i1); break;
        case 3: p2p_launch64_t<3>(P, st, wf, i0, i1); break;
        case 4: p2p_launch64_t<4>(P, st, wf, i0, i1); break;
        case 5: p2p_launch64_t<5>(P, st, wf, i0, i1); break;
        case 6: p2p_launch64_t<6>(P, st, wf, i0, i1); break;
        case 7: p2p_launch64_t<7>(P, st, wf, i0, i1); break;
        default: p2p_launch64_t<8>(P, st, wf, i0, i1); break;
    }
}

}  // namespace fmm
