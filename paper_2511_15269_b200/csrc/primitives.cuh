// primitives.cuh -- hand-written device-wide primitives used by the plan phase:
// exclusive scan (3-phase, recursive over block sums) and a stable LSD radix sort of (key, value) pairs.
#pragma once
#include "internal.cuh"

namespace fmm {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

template <typename V>
struct PtrLoad {
    const V* p;
    __device__ V operator()(int64_t i) const { return p[i]; }
};

template <typename V>
__device__ inline V block_exclusive_scan(V x, V* total, V* smem /* >= 33 entries */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    V incl = x;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        V y = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += y;
    }
    if (lane == 31) smem[w] = incl;
    __syncthreads();
    if (w == 0) {
        V v = (lane < (int)(blockDim.x >> 5)) ? smem[lane] : V(0);
        V inc2 = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            V y = __shfl_up_sync(0xffffffffu, inc2, d);
            if (lane >= d) inc2 += y;
        }
        smem[lane] = inc2 - v;  // exclusive warp offsets
        if (lane == 31) smem[32] = inc2;
    }
    __syncthreads();
    V res = incl - x + smem[w];
    if (total) *total = smem[32];
    __syncthreads();
    return res;
}

template <typename V, typename LoadF>
__global__ void __launch_bounds__(SCAN_THREADS) scan_reduce_k(LoadF load, V* block_sums, int64_t n) {
    __shared__ V sm[33];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    V s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i)
        if (base + i < n) s += load(base + i);
    V tot;
    block_exclusive_scan<V>(s, &tot, sm);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = tot;
}

template <typename V, typename LoadF>
__global__ void __launch_bounds__(SCAN_THREADS) scan_apply_k(LoadF load, V* out, const V* block_offs, int64_t n) {
    __shared__ V sm[33];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    V v[SCAN_ITEMS];
    V s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        v[i] = (base + i < n) ? load(base + i) : V(0);
        s += v[i];
    }
    V off = block_exclusive_scan<V>(s, nullptr, sm) + (block_offs ? block_offs[blockIdx.x] : V(0));
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        if (base + i < n) out[base + i] = off;
        off += v[i];
    }
}

// Exclusive scan of load(0..n-1) into out[0..n-1].  scratch must hold scan_scratch_elems(n) elements of V.
inline int64_t scan_scratch_elems(int64_t n) {
    int64_t tot = 0;
    while (n > 1) {
        n = (n + SCAN_TILE - 1) / SCAN_TILE;
        tot += n + 1;
        if (n == 1) break;
    }
    return tot + 2;
}

template <typename V, typename LoadF>
void exclusive_scan(LoadF load, V* out, int64_t n, V* scratch, cudaStream_t st) {
    if (n <= 0) return;
    const int64_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (nb == 1) {
        scan_apply_k<V, LoadF><<<1, SCAN_THREADS, 0, st>>>(load, out, nullptr, n);
        FMM_CUDA_CHECK(cudaGetLastError());
        return;
    }
    scan_reduce_k<V, LoadF><<<(unsigned)nb, SCAN_THREADS, 0, st>>>(load, scratch, n);
    FMM_CUDA_CHECK(cudaGetLastError());
    exclusive_scan<V, PtrLoad<V>>(PtrLoad<V>{scratch}, scratch, nb, scratch + nb + 1, st);  // in place
    scan_apply_k<V, LoadF><<<(unsigned)nb, SCAN_THREADS, 0, st>>>(load, out, scratch, n);
    FMM_CUDA_CHECK(cudaGetLastError());
}

// ------------------------------------------------------------------------------------------------
// Stable LSD radix sort, 8 bits per pass, (KeyT key, int32 value).
// ------------------------------------------------------------------------------------------------
constexpr int RS_WARPS = 8;
constexpr int RS_CHUNKS = 16;                         // 32-item chunks per warp
constexpr int RS_TILE = RS_WARPS * RS_CHUNKS * 32;    // items per block

template <typename KeyT>
__global__ void __launch_bounds__(RS_WARPS * 32) radix_hist_k(const KeyT* keys, int64_t n, int shift, int32_t* hist, int nblk) {
    __shared__ int32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * RS_TILE;
    for (int i = threadIdx.x; i < RS_TILE; i += RS_WARPS * 32) {
        const int64_t g = base + i;
        if (g < n) atomicAdd(&h[(int)((keys[g] >> shift) & 0xff)], 1);
    }
    __syncthreads();
    hist[(int64_t)threadIdx.x * nblk + blockIdx.x] = h[threadIdx.x];
}

template <typename KeyT>
__global__ void __launch_bounds__(RS_WARPS * 32) radix_scatter_k(const KeyT* keys_in, const int32_t* vals_in, KeyT* keys_out,
                                                                  int32_t* vals_out, int64_t n, int shift,
                                                                  const int32_t* hist_scanned, int nblk) {
    __shared__ int32_t wh[RS_WARPS][256];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < RS_WARPS * 256; i += RS_WARPS * 32) (&wh[0][0])[i] = 0;
    __syncthreads();
    const int64_t wbase = (int64_t)blockIdx.x * RS_TILE + (int64_t)w * RS_CHUNKS * 32;
    for (int c = 0; c < RS_CHUNKS; ++c) {
        const int64_t g = wbase + c * 32 + lane;
        if (g < n) atomicAdd(&wh[w][(int)((keys_in[g] >> shift) & 0xff)], 1);
    }
    __syncthreads();
    {
        const int d = threadIdx.x;  // 256 threads <-> 256 digits
        int32_t run = hist_scanned[(int64_t)d * nblk + blockIdx.x];
        for (int ww = 0; ww < RS_WARPS; ++ww) {
            const int32_t t = wh[ww][d];
            wh[ww][d] = run;
            run += t;
        }
    }
    __syncthreads();
    for (int c = 0; c < RS_CHUNKS; ++c) {
        const int64_t g = wbase + c * 32 + lane;
        const bool valid = g < n;
        const unsigned act = __ballot_sync(0xffffffffu, valid);
        if (valid) {
            const KeyT k = keys_in[g];
            const int d = (int)((k >> shift) & 0xff);
            const unsigned grp = __match_any_sync(act, d);
            const int leader = __ffs(grp) - 1;
            int32_t basepos = 0;
            if (lane == leader) {
                basepos = wh[w][d];
                wh[w][d] = basepos + __popc(grp);
            }
            basepos = __shfl_sync(grp, basepos, leader);
            const int32_t dest = basepos + __popc(grp & ((1u << lane) - 1u));
            keys_out[dest] = k;
            vals_out[dest] = vals_in[g];
        }
        __syncwarp();
    }
}

// sorts n pairs by the low `bits` bits of the key; result ends in (keys_a, vals_a) if the number of passes is even,
// else in (keys_b, vals_b): returns 0 or 1 accordingly.  hist: 256*nblk+1 int32 (+ scan scratch).
template <typename KeyT>
int radix_sort_pairs(KeyT* keys_a, int32_t* vals_a, KeyT* keys_b, int32_t* vals_b, int64_t n, int bits, int32_t* hist,
                     int32_t* scan_scratch, cudaStream_t st) {
    const int nblk = (int)((n + RS_TILE - 1) / RS_TILE);
    int cur = 0;
    for (int shift = 0; shift < bits; shift += 8) {
        KeyT* ki = cur ? keys_b : keys_a;
        KeyT* ko = cur ? keys_a : keys_b;
        int32_t* vi = cur ? vals_b : vals_a;
        int32_t* vo = cur ? vals_a : vals_b;
        radix_hist_k<KeyT><<<nblk, RS_WARPS * 32, 0, st>>>(ki, n, shift, hist, nblk);
        FMM_CUDA_CHECK(cudaGetLastError());
        exclusive_scan<int32_t, PtrLoad<int32_t>>(PtrLoad<int32_t>{hist}, hist, (int64_t)256 * nblk, scan_scratch, st);
        radix_scatter_k<KeyT><<<nblk, RS_WARPS * 32, 0, st>>>(ki, vi, ko, vo, n, shift, hist, nblk);
        FMM_CUDA_CHECK(cudaGetLastError());
        cur ^= 1;
    }
    return cur;
}

}  // namespace fmm
