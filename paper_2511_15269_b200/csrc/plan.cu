// plan.cu -- device-side hierarchy (median-split 2^s-tree) and interaction-list construction.
//
// Hierarchy: PAPER.md:40-43 and Listing 2.  The paper re-partitions every box with
// argpartition at each of the s*L sub-splits; here each axis is radix-sorted ONCE by (coordinate, input index)
// and the four orderings (x, y, z, index) are then stably partitioned per sub-split, so that
//   * the tight bounding box of a node is read off the ends of its three sorted segments (no reduction pass),
//   * the median is a direct lookup in the segment of the split axis,
//   * ties are resolved by the total order (coordinate, input index) (reading S4),
//   * leaves end up in ascending input index (final jnp.sort of Listing 2).
// Which half receives the odd particle follows Listing 2's padding (DESIGN.md rule T3): with n_d the padded
// row length at sub-depth d, the upper child takes the last floor(n_d/2) particles.
//
// Lists: PAPER.md:72-74 with criterion (4) PAPER.md:68-70, evaluated in non-contracted IEEE fp64.
#include <algorithm>
#include <climits>

#include "primitives.cuh"

namespace fmm {
namespace {

// ---------------------------------------------------------------------------------------------- keys
__device__ inline uint32_t order_key(float x) {
    if (x == 0.0f) x = 0.0f;  // -0 -> +0
    const uint32_t b = __float_as_uint(x);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ inline uint64_t order_key(double x) {
    if (x == 0.0) x = 0.0;
    const uint64_t b = (uint64_t)__double_as_longlong(x);
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}

template <typename T, typename KeyT>
__global__ void make_keys_k(const T* pos, int64_t N, int axis, KeyT* keys, int32_t* vals, int* bad) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const T x = pos[3 * i + axis];
    if (!isfinite(x)) *bad = 1;
    keys[i] = order_key(x);
    vals[i] = (int32_t)i;
}

__global__ void invert_perm_k(const int32_t* ord, int32_t* rank, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) rank[ord[i]] = (int32_t)i;
}

__global__ void iota_k(int32_t* a, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) a[i] = (int32_t)i;
}

// ---------------------------------------------------------------------------------------------- tree rounds
struct OrdPtrs {
    const int32_t* o[4];  // x, y, z, index orderings (particle ids, segmented by node)
};

// one thread per node of sub-depth d
template <typename T>
__global__ void node_k(const T* pos, OrdPtrs ord, const int32_t* rank0, const int32_t* rank1, const int32_t* rank2,
                       const int32_t* nstart, const int32_t* ncnt, int64_t nnodes, int64_t n_d, int is_level, int is_last,
                       int64_t box_off, int32_t* box_start, int32_t* box_count, T* box_lo, T* box_hi,
                       int32_t* naxis, int32_t* npivot, int32_t* nstart2, int32_t* ncnt2) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nnodes) return;
    const int32_t st = nstart[j], c = ncnt[j];
    T lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    if (c > 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = pos[3 * (int64_t)ord.o[a][st] + a];
            hi[a] = pos[3 * (int64_t)ord.o[a][st + c - 1] + a];
        }
    }
    if (is_level) {
        const int64_t g = box_off + j;
        box_start[g] = st;
        box_count[g] = c;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            box_lo[3 * g + a] = lo[a];
            box_hi[3 * g + a] = hi[a];
        }
    }
    if (is_last) return;
    int32_t n_up = (int32_t)(n_d / 2);
    if (n_up > c) n_up = c;
    const int32_t n_lo = c - n_up;
    int axis = 0;
    if (c > 0) {  // longest extent in fp64, ties -> lowest axis (first maximum of jnp.argmax)
        const double e0 = (double)hi[0] - (double)lo[0], e1 = (double)hi[1] - (double)lo[1], e2 = (double)hi[2] - (double)lo[2];
        double eb = e0;
        if (e1 > eb) { axis = 1; eb = e1; }
        if (e2 > eb) { axis = 2; }
    }
    int32_t pivot = INT_MAX;
    if (n_up > 0) {
        const int32_t pt = ord.o[axis][st + n_lo];
        pivot = (axis == 0 ? rank0 : axis == 1 ? rank1 : rank2)[pt];
    }
    naxis[j] = axis;
    npivot[j] = pivot;
    nstart2[2 * j] = st;
    ncnt2[2 * j] = n_lo;
    nstart2[2 * j + 1] = st + n_lo;
    ncnt2[2 * j + 1] = n_up;
}

__global__ void pflag_k(const int32_t* pnode, const int32_t* rank0, const int32_t* rank1, const int32_t* rank2,
                        const int32_t* naxis, const int32_t* npivot, uint8_t* pflag, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int32_t nd = pnode[i];
    const int ax = naxis[nd];
    const int32_t r = (ax == 0 ? rank0 : ax == 1 ? rank1 : rank2)[i];
    pflag[i] = r >= npivot[nd] ? 1 : 0;
}

struct FlagLoad {
    const uint8_t* pflag;
    const int32_t* ord;
    int64_t N;
    __device__ int32_t operator()(int64_t i) const { return i < N ? (int32_t)pflag[ord[i]] : 0; }
};

__global__ void partition_k(const int32_t* ord_in, int32_t* ord_out, const int32_t* F, const uint8_t* pflag, const int32_t* pnode,
                            const int32_t* nstart, const int32_t* nstart2, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int32_t pt = ord_in[i];
    const int32_t nd = pnode[pt];
    const int32_t s0 = nstart[nd];
    const int32_t ups = F[i] - F[s0];  // flagged elements of this node before position i
    int32_t dest;
    if (pflag[pt]) dest = nstart2[2 * nd + 1] + ups;
    else dest = nstart2[2 * nd] + ((int32_t)i - s0) - ups;
    ord_out[dest] = pt;
}

// ---- the four orderings (x, y, z, index) of one sub-split in ONE launch per phase (blockIdx.y = ordering): the rounds are
// latency-bound (150 launches of ~10 us at N = 1M when every ordering has its own scan and partition kernels)
struct Ord4 {
    const int32_t* in[4];
    int32_t* out[4];
};
__global__ void __launch_bounds__(SCAN_THREADS) flag4_reduce_k(const uint8_t* pflag, Ord4 o, int64_t N, int32_t* block_sums, int64_t nb) {
    __shared__ int32_t sm[33];
    const int32_t* ord = o.in[blockIdx.y];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    int32_t s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i)
        if (base + i < N) s += pflag[ord[base + i]];
    int32_t tot;
    block_exclusive_scan<int32_t>(s, &tot, sm);
    if (threadIdx.x == 0) block_sums[blockIdx.y * nb + blockIdx.x] = tot;
}
// exclusive scan of the nb <= SCAN_TILE block sums of each ordering, one block per ordering, in place
__global__ void __launch_bounds__(SCAN_THREADS) flag4_sums_k(int32_t* block_sums, int64_t nb) {
    __shared__ int32_t sm[33];
    int32_t* b = block_sums + blockIdx.y * nb;
    const int64_t base = (int64_t)threadIdx.x * SCAN_ITEMS;
    int32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = base + i < nb ? b[base + i] : 0; s += v[i]; }
    int32_t off = block_exclusive_scan<int32_t>(s, nullptr, sm);
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { if (base + i < nb) b[base + i] = off; off += v[i]; }
}
// F[y][i] = number of flagged particles before position i of ordering y (i = 0..N; F has N + 1 entries per ordering)
__global__ void __launch_bounds__(SCAN_THREADS) flag4_apply_k(const uint8_t* pflag, Ord4 o, int64_t N, const int32_t* block_offs, int64_t nb, int32_t* F) {
    __shared__ int32_t sm[33];
    const int32_t* ord = o.in[blockIdx.y];
    int32_t* Fy = F + blockIdx.y * (N + 1);
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    int32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = base + i < N ? (int32_t)pflag[ord[base + i]] : 0; s += v[i]; }
    int32_t off = block_exclusive_scan<int32_t>(s, nullptr, sm) + block_offs[blockIdx.y * nb + blockIdx.x];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { if (base + i <= N) Fy[base + i] = off; off += v[i]; }
}
__global__ void partition4_k(Ord4 o, const int32_t* F, const uint8_t* pflag, const int32_t* pnode, const int32_t* nstart, const int32_t* nstart2, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int32_t* Fy = F + blockIdx.y * (N + 1);
    const int32_t pt = o.in[blockIdx.y][i];
    const int32_t nd = pnode[pt];
    const int32_t s0 = nstart[nd];
    const int32_t ups = Fy[i] - Fy[s0];  // flagged elements of this node before position i
    int32_t dest;
    if (pflag[pt]) dest = nstart2[2 * nd + 1] + ups;
    else dest = nstart2[2 * nd] + ((int32_t)i - s0) - ups;
    o.out[blockIdx.y][dest] = pt;
}

__global__ void pnode_update_k(int32_t* pnode, const uint8_t* pflag, int64_t N) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) pnode[i] = 2 * pnode[i] + pflag[i];
}

// ---------------------------------------------------------------------------------------------- geometry (rule T6)
template <typename T>
__global__ void geometry_k(const T* lo, const T* hi, const int32_t* cnt, int64_t off, int64_t nb, int64_t off_parent, int s,
                           double* ctr, double* rad, T* scale) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const int64_t g = off + b;
    double d[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double l = (double)lo[3 * g + a], h = (double)hi[3 * g + a];
        ctr[3 * g + a] = __dmul_rn(0.5, __dadd_rn(l, h));
        d[a] = __dsub_rn(h, l);
    }
    const double r = __dmul_rn(0.5, __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]))));
    rad[g] = r;
    // expansion length scale: the radius, inherited from the parent for point-like boxes (any positive value is valid)
    T sc = (T)r;
    if (!(sc > (T)0)) sc = (off_parent >= 0) ? scale[off_parent + (b >> s)] : (T)1;
    scale[g] = sc;
    (void)cnt;
}

template <typename T>
__global__ void gather_pos_k(const T* pos, const int32_t* perm, T* pos_tree, int64_t N) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int64_t i = perm[k];
    pos_tree[3 * k] = pos[3 * i];
    pos_tree[3 * k + 1] = pos[3 * i + 1];
    pos_tree[3 * k + 2] = pos[3 * i + 2];
}

// P2P source-group slots (fp32): particle i of leaf l -> 4 * (l * G + i / 4) + (i & 3); one warp per leaf
__global__ void srcg_init_k(float* srcg, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) srcg[i] = (i & 15) < 12 ? 1e18f : 0.f;  // group = (-x[4], -y[4], -z[4], q[4])
}
__global__ void src_slot_k(const int32_t* leaf_start, const int32_t* leaf_cnt, int64_t n_leaves, int G, int32_t* slot) {
    const int64_t leaf = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (leaf >= n_leaves) return;
    const int st = leaf_start[leaf], c = leaf_cnt[leaf];
    for (int i = threadIdx.x & 31; i < c; i += 32) slot[st + i] = (int32_t)(4 * (leaf * G + (i >> 2)) + (i & 3));
}

inline unsigned nblocks(int64_t n, int t) { return (unsigned)((n + t - 1) / t); }

template <typename T, typename KeyT>
void build_tree_t(Plan& P, const T* pos, cudaStream_t st) {
    const int64_t N = P.N;
    const int dmax = P.s * P.L;
    const int64_t n_leaves = (int64_t)1 << dmax;
    cudaEvent_t e0, e1, e2;
    FMM_CUDA_CHECK(cudaEventCreate(&e0));
    FMM_CUDA_CHECK(cudaEventCreate(&e1));
    FMM_CUDA_CHECK(cudaEventCreate(&e2));
    FMM_CUDA_CHECK(cudaEventRecord(e0, st));

    DevBuf<KeyT> keys_a, keys_b;
    DevBuf<int32_t> vals_b, hist, scan_scratch, rank[3], ordA[4], ordB[4], pnode, F;
    DevBuf<uint8_t> pflag;
    DevBuf<int> bad;
    keys_a.alloc(N); keys_b.alloc(N); vals_b.alloc(N);
    const int nblk = (int)((N + RS_TILE - 1) / RS_TILE);
    hist.alloc((size_t)256 * nblk + 1);
    scan_scratch.alloc((size_t)std::max(scan_scratch_elems((int64_t)256 * nblk), scan_scratch_elems(N + 1)));
    for (int a = 0; a < 3; ++a) rank[a].alloc(N);
    for (int a = 0; a < 4; ++a) { ordA[a].alloc(N); ordB[a].alloc(N); }
    const int64_t nb_scan = (N + 1 + SCAN_TILE - 1) / SCAN_TILE;
    const bool fused4 = nb_scan <= SCAN_TILE;  // the block sums of one ordering fit one scan block (N <= 4.19M); else one ordering at a time
    DevBuf<int32_t> sums4;
    if (fused4) sums4.alloc((size_t)4 * nb_scan);
    pnode.alloc(N); F.alloc(fused4 ? 4 * (N + 1) : N + 1); pflag.alloc(N);
    bad.alloc(1);
    FMM_CUDA_CHECK(cudaMemsetAsync(bad.p, 0, sizeof(int), st));

    // 1. three stable radix sorts by (coordinate, input index)
    for (int a = 0; a < 3; ++a) {
        make_keys_k<T, KeyT><<<nblocks(N, 256), 256, 0, st>>>(pos, N, a, keys_a.p, ordA[a].p, bad.p);
        FMM_CUDA_CHECK(cudaGetLastError());
        const int where = radix_sort_pairs<KeyT>(keys_a.p, ordA[a].p, keys_b.p, vals_b.p, N, (int)sizeof(KeyT) * 8, hist.p, scan_scratch.p, st);
        if (where == 1) FMM_CUDA_CHECK(cudaMemcpyAsync(ordA[a].p, vals_b.p, N * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        invert_perm_k<<<nblocks(N, 256), 256, 0, st>>>(ordA[a].p, rank[a].p, N);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    iota_k<<<nblocks(N, 256), 256, 0, st>>>(ordA[3].p, N);
    FMM_CUDA_CHECK(cudaGetLastError());
    int h_bad = 0;
    FMM_CUDA_CHECK(cudaMemcpyAsync(&h_bad, bad.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    if (h_bad) {
        set_error("positions contain non-finite values");
        throw CudaFail{FMM_ERR_INVALID_ARG};
    }
    FMM_CUDA_CHECK(cudaEventRecord(e1, st));

    // 2. s*L rounds of stable partition
    P.box_start.alloc(P.n_boxes); P.box_count.alloc(P.n_boxes);
    P.box_lo.alloc(P.n_boxes * 3 * sizeof(T)); P.box_hi.alloc(P.n_boxes * 3 * sizeof(T));
    DevBuf<int32_t> nstart[2], ncnt[2], naxis, npivot;
    for (int k = 0; k < 2; ++k) { nstart[k].alloc(n_leaves); ncnt[k].alloc(n_leaves); }
    naxis.alloc(n_leaves); npivot.alloc(n_leaves);
    {
        const int32_t z = 0, n32 = (int32_t)N;
        FMM_CUDA_CHECK(cudaMemcpyAsync(nstart[0].p, &z, 4, cudaMemcpyHostToDevice, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(ncnt[0].p, &n32, 4, cudaMemcpyHostToDevice, st));
        FMM_CUDA_CHECK(cudaMemsetAsync(pnode.p, 0, N * sizeof(int32_t), st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    }
    int32_t *oa[4], *ob[4];
    for (int a = 0; a < 4; ++a) { oa[a] = ordA[a].p; ob[a] = ordB[a].p; }
    int64_t n_d = N;
    int cur = 0;
    for (int d = 0; d <= dmax; ++d) {
        const int64_t nnodes = (int64_t)1 << d;
        const int is_level = (d % P.s == 0) ? 1 : 0;
        const int is_last = (d == dmax) ? 1 : 0;
        OrdPtrs op;
        for (int a = 0; a < 4; ++a) op.o[a] = oa[a];
        node_k<T><<<nblocks(nnodes, 128), 128, 0, st>>>(pos, op, rank[0].p, rank[1].p, rank[2].p, nstart[cur].p, ncnt[cur].p, nnodes, n_d,
                                                        is_level, is_last, is_level ? P.level_off[d / P.s] : 0, P.box_start.p, P.box_count.p,
                                                        (T*)P.box_lo.p, (T*)P.box_hi.p, naxis.p, npivot.p, nstart[cur ^ 1].p, ncnt[cur ^ 1].p);
        FMM_CUDA_CHECK(cudaGetLastError());
        if (is_last) break;
        pflag_k<<<nblocks(N, 256), 256, 0, st>>>(pnode.p, rank[0].p, rank[1].p, rank[2].p, naxis.p, npivot.p, pflag.p, N);
        FMM_CUDA_CHECK(cudaGetLastError());
        if (fused4) {
            Ord4 o4;
            for (int a = 0; a < 4; ++a) { o4.in[a] = oa[a]; o4.out[a] = ob[a]; }
            flag4_reduce_k<<<dim3((unsigned)nb_scan, 4), SCAN_THREADS, 0, st>>>(pflag.p, o4, N, sums4.p, nb_scan);
            flag4_sums_k<<<dim3(1, 4), SCAN_THREADS, 0, st>>>(sums4.p, nb_scan);
            flag4_apply_k<<<dim3((unsigned)nb_scan, 4), SCAN_THREADS, 0, st>>>(pflag.p, o4, N, sums4.p, nb_scan, F.p);
            partition4_k<<<dim3(nblocks(N, 256), 4), 256, 0, st>>>(o4, F.p, pflag.p, pnode.p, nstart[cur].p, nstart[cur ^ 1].p, N);
            FMM_CUDA_CHECK(cudaGetLastError());
            for (int a = 0; a < 4; ++a) std::swap(oa[a], ob[a]);
        } else
            for (int a = 0; a < 4; ++a) {
                exclusive_scan<int32_t, FlagLoad>(FlagLoad{pflag.p, oa[a], N}, F.p, N + 1, scan_scratch.p, st);
                partition_k<<<nblocks(N, 256), 256, 0, st>>>(oa[a], ob[a], F.p, pflag.p, pnode.p, nstart[cur].p, nstart[cur ^ 1].p, N);
                FMM_CUDA_CHECK(cudaGetLastError());
                std::swap(oa[a], ob[a]);
            }
        pnode_update_k<<<nblocks(N, 256), 256, 0, st>>>(pnode.p, pflag.p, N);
        FMM_CUDA_CHECK(cudaGetLastError());
        n_d = (n_d + 1) / 2;
        cur ^= 1;
    }
    P.max_leaf = (int)n_d;
    P.perm.alloc(N);
    FMM_CUDA_CHECK(cudaMemcpyAsync(P.perm.p, oa[3], N * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));

    // 3. geometry, top-down (scale inherits from the parent)
    P.box_ctr.alloc(P.n_boxes * 3); P.box_rad.alloc(P.n_boxes); P.box_scale.alloc(P.n_boxes * sizeof(T));
    for (int l = 0; l <= P.L; ++l) {
        const int64_t nb = (int64_t)1 << (P.s * l);
        geometry_k<T><<<nblocks(nb, 128), 128, 0, st>>>((const T*)P.box_lo.p, (const T*)P.box_hi.p, P.box_count.p, P.level_off[l], nb,
                                                        l > 0 ? P.level_off[l - 1] : -1, P.s, P.box_ctr.p, P.box_rad.p, (T*)P.box_scale.p);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    if (sizeof(T) == 4) {
        P.src_G = (P.max_leaf + 3) / 4;
        if (4 * (n_leaves * P.src_G + 1) > 0x7fffffffll) {
            set_error("too many P2P source groups for 32-bit slots");
            throw CudaFail{FMM_ERR_UNSUPPORTED};
        }
        P.src_slot.alloc(N);
        P.srcg.alloc((size_t)n_leaves * P.src_G * 16);
        // pad slots: zero charge, parked at x = y = z = -1e18 (stored negated), far from every real particle and from the parked
        // target slots at +1e18, so that their distance is never zero and no mask is needed for them
        srcg_init_k<<<nblocks((int64_t)P.srcg.n, 256), 256, 0, st>>>(P.srcg.p, (int64_t)P.srcg.n);
        FMM_CUDA_CHECK(cudaGetLastError());
        src_slot_k<<<nblocks(n_leaves * 32, 128), 128, 0, st>>>(P.box_start.p + P.level_off[P.L], P.box_count.p + P.level_off[P.L], n_leaves,
                                                               P.src_G, P.src_slot.p);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    P.pos_tree.alloc(N * 3 * sizeof(T));
    gather_pos_k<T><<<nblocks(N, 256), 256, 0, st>>>(pos, P.perm.p, (T*)P.pos_tree.p, N);
    FMM_CUDA_CHECK(cudaGetLastError());
    FMM_CUDA_CHECK(cudaEventRecord(e2, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    float ms1 = 0, ms2 = 0;
    cudaEventElapsedTime(&ms1, e0, e1);
    cudaEventElapsedTime(&ms2, e1, e2);
    P.plan_ms[0] = ms1;
    P.plan_ms[1] = ms2;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(e2);
}

// ---------------------------------------------------------------------------------------------- lists
// eq. (4) PAPER.md:68-70 (rule L1): R + theta*r < theta*d, strict, IEEE fp64 without contraction.
// (ctr_a, rad_a) / (ctr_b, rad_b): geometry arrays of the hierarchy box a / box b belongs to (the same arrays for one hierarchy)
__device__ inline bool admissible2(const double* ctr, const double* rad, int64_t ga, const double* ctr_b, const double* rad_b, int64_t gb, double theta) {
    const double ra = rad[ga], rb = rad_b[gb];
    const double R = fmax(ra, rb), r = fmin(ra, rb);
    const double dx = __dsub_rn(ctr[3 * ga], ctr_b[3 * gb]);
    const double dy = __dsub_rn(ctr[3 * ga + 1], ctr_b[3 * gb + 1]);
    const double dz = __dsub_rn(ctr[3 * ga + 2], ctr_b[3 * gb + 2]);
    const double d = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
    return __dadd_rn(R, __dmul_rn(theta, r)) < __dmul_rn(theta, d);
}
__device__ inline bool admissible(const double* ctr, const double* rad, int64_t ga, int64_t gb, double theta) {
    const double ra = rad[ga], rb = rad[gb];
    const double R = fmax(ra, rb), r = fmin(ra, rb);
    const double dx = __dsub_rn(ctr[3 * ga], ctr[3 * gb]);
    const double dy = __dsub_rn(ctr[3 * ga + 1], ctr[3 * gb + 1]);
    const double dz = __dsub_rn(ctr[3 * ga + 2], ctr[3 * gb + 2]);
    const double d = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
    return __dadd_rn(R, __dmul_rn(theta, r)) < __dmul_rn(theta, d);
}

struct ExpandArgs {
    const int32_t *ftgt, *fsrc;  // failing pairs of the parent level (level-local indices), sorted by (tgt, src)
    const int64_t* foff;         // CSR offsets of the failing pairs by parent target
    int64_t nfail;
    int s;
    int64_t off_child;           // global id offset of the child level
    const int32_t* box_count;
    const double *ctr, *rad;
    double theta;
};

__device__ inline void expand_decode(const ExpandArgs& A, int64_t idx, int64_t& pos, int32_t& t, int32_t& sc) {
    const int nch = 1 << A.s, nch2 = nch * nch;
    const int64_t e = idx / nch2;
    const int ij = (int)(idx - e * nch2);
    const int i = ij >> A.s, j = ij & (nch - 1);
    const int32_t a = A.ftgt[e], b = A.fsrc[e];
    const int64_t row0 = A.foff[a], rowlen = A.foff[a + 1] - row0;
    pos = row0 * nch2 + (int64_t)i * (rowlen * nch) + (e - row0) * nch + j;
    t = a * nch + i;
    sc = b * nch + j;
}

// codes: 0 = dropped (empty box), 1 = weak (admissible), 2 = fail (to be refined / strong)
__global__ void expand_classify_k(ExpandArgs A, uint8_t* codes) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t total = A.nfail << (2 * A.s);
    if (idx >= total) return;
    int64_t pos; int32_t t, sc;
    expand_decode(A, idx, pos, t, sc);
    const int64_t gt = A.off_child + t, gs = A.off_child + sc;
    uint8_t code = 0;
    if (A.box_count[gt] > 0 && A.box_count[gs] > 0) code = admissible(A.ctr, A.rad, gt, gs, A.theta) ? 1 : 2;
    codes[pos] = code;
}

struct CodeLoad {
    const uint8_t* codes;
    int64_t n;
    __device__ unsigned long long operator()(int64_t i) const {
        if (i >= n) return 0ull;
        const uint8_t c = codes[i];
        return c == 1 ? 1ull : (c == 2 ? (1ull << 32) : 0ull);
    }
};

__global__ void expand_compact_k(ExpandArgs A, const uint8_t* codes, const unsigned long long* S, int32_t* wtgt, int32_t* wsrc,
                                 int32_t* ftgt2, int32_t* fsrc2) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t total = A.nfail << (2 * A.s);
    if (idx >= total) return;
    int64_t pos; int32_t t, sc;
    expand_decode(A, idx, pos, t, sc);
    const uint8_t c = codes[pos];
    const unsigned long long sv = S[pos];
    if (c == 1) {
        const int64_t o = (int64_t)(sv & 0xffffffffull);
        wtgt[o] = (int32_t)(A.off_child + t);
        wsrc[o] = (int32_t)(A.off_child + sc);
    } else if (c == 2) {
        const int64_t o = (int64_t)(sv >> 32);
        ftgt2[o] = t;
        fsrc2[o] = sc;
    }
}

// row offsets of the child level: thread per child target (+1 for the end)
__global__ void expand_offsets_k(ExpandArgs A, const unsigned long long* S, int64_t nb_child, int64_t total, int64_t weak_base,
                                 int64_t* weak_off_global, int64_t* foff2) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t > nb_child) return;
    int64_t base;
    if (t == nb_child) base = total;
    else {
        const int nch = 1 << A.s;
        const int64_t a = t >> A.s;
        const int i = (int)(t & (nch - 1));
        const int64_t row0 = A.foff[a], rowlen = A.foff[a + 1] - row0;
        base = row0 * nch * nch + (int64_t)i * rowlen * nch;
    }
    const unsigned long long sv = S[base];
    weak_off_global[A.off_child + t] = weak_base + (int64_t)(sv & 0xffffffffull);
    foff2[t] = (int64_t)(sv >> 32);
}

// strong_touch[e] = 1 iff the tight bounding boxes of the target leaf and the source leaf of entry e touch or overlap (comparisons
// in the plan's dtype): only then can a target coincide with a source (reading S3)
template <typename T>
__global__ void strong_touch_k(const int64_t* soff, const int32_t* ssrc, const T* tlo, const T* thi, const T* slo, const T* shi, int64_t n_leaves, uint8_t* touch) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_leaves) return;
    const T a0 = tlo[3 * t], a1 = tlo[3 * t + 1], a2 = tlo[3 * t + 2], b0 = thi[3 * t], b1 = thi[3 * t + 1], b2 = thi[3 * t + 2];
    for (int64_t e = soff[t]; e < soff[t + 1]; ++e) {
        const int64_t s = ssrc[e];
        // fp32: pairs with r^2 < FLT_MIN count as coincident (reading S3), so boxes closer than sqrt(FLT_MIN) ~ 1.08e-19 along every
        // axis are flagged as well (tol is conservative); fp64: exact comparisons
        const T tol = sizeof(T) == 4 ? (T)2e-19 : (T)0;
        const bool hit = a0 - shi[3 * s] <= tol && slo[3 * s] - b0 <= tol && a1 - shi[3 * s + 1] <= tol && slo[3 * s + 1] - b1 <= tol &&
                         a2 - shi[3 * s + 2] <= tol && slo[3 * s + 2] - b2 <= tol;
        touch[e] = hit ? 1 : 0;
    }
}

// out[0] = number of particle pairs of the P2P stage, out[1] = sum over non-empty target leaves of their source particles
__global__ void count_p2p_k(const int64_t* soff, const int32_t* ssrc, const int32_t* leaf_cnt, const int32_t* src_cnt, int64_t n_leaves, unsigned long long* out) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long acc = 0, ssum = 0;
    if (t < n_leaves && leaf_cnt[t] > 0) {
        for (int64_t e = soff[t]; e < soff[t + 1]; ++e) ssum += (unsigned long long)src_cnt[ssrc[e]];
        acc = ssum * (unsigned long long)leaf_cnt[t];
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, d);
        ssum += __shfl_xor_sync(0xffffffffu, ssum, d);
    }
    if ((threadIdx.x & 31) == 0 && acc) {
        atomicAdd(out, acc);
        atomicAdd(out + 1, ssum);
    }
}

// P2P work items: the strong list of a target leaf is cut into segments of at most `budget` source particles (whole source
// leaves; a segment closes as soon as it has reached the budget), so that one warp never owns more than about twice the
// average work even when a few leaves have very long lists (clustered inputs).  Pass 1 (items == nullptr) counts the segments
// of every leaf, pass 2 writes them at seg_off[leaf].
struct SegLoad {
    const int32_t* p;
    int64_t n;
    __device__ int64_t operator()(int64_t i) const { return i < n ? (int64_t)p[i] : 0; }
};
__global__ void p2p_segments_k(const int64_t* soff, const int32_t* ssrc, const int32_t* leaf_start, const int32_t* leaf_cnt, const int32_t* src_cnt, int64_t n_leaves, int64_t budget,
                               int32_t* nseg, const int64_t* seg_off, P2PItem* items, int* any_multi) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_leaves) return;
    int n = 0;
    if (leaf_cnt[t] > 0) {
        const int total = items ? nseg[t] : 0;
        int64_t acc = 0, e0 = soff[t];
        const int64_t eend = soff[t + 1];
        for (int64_t e = e0; e < eend; ++e) {
            acc += src_cnt[ssrc[e]];
            if (acc >= budget || e + 1 == eend) {
                if (items) items[seg_off[t] + n] = P2PItem{leaf_start[t], leaf_cnt[t], e0, total > 1 ? ~(e + 1) : e + 1};
                ++n;
                acc = 0;
                e0 = e + 1;
            }
        }
    }
    if (!items) {
        nseg[t] = n;
        if (n > 1) *any_multi = 1;
    }
}

// ---- level-marching (cross-level) lists, reading S9: steps (lt, ls) = (0,0), (0,1), (1,1), (1,2), ..., (L,L).
// Failing pairs (target box on level lt, source box on level ls; level-local indices) are refined on ONE side per step:
// the sources when lt == ls ("if equal, increase the source level"), else the targets.  A source box is therefore
// never coarser than its target box, which the split schedule of evaluate.cu relies on (the leaf-level M2L reads only
// leaf-level multipoles and may run beside the M2M pass).  Invariant: for a fixed target the sources appear in ascending order, so a
// stable sort by target at the end gives the canonical CSR form (L4) that is compared bit by bit with the oracle.
struct MarchArgs {
    const int32_t *ftgt, *fsrc;
    int64_t nfail;
    int s;
    int refine_src;                 // 1: candidates (t, s * nch + c) ; 0: candidates (t * nch + c, s)
    int64_t off_t, off_s;           // global id offsets of the candidates' levels
    const int32_t* box_count;       // target hierarchy
    const double *ctr, *rad;
    const int32_t* count_s;         // source hierarchy (the same arrays when sources and targets share one hierarchy)
    const double *ctr_s, *rad_s;
    double theta;
};
__device__ inline void march_decode(const MarchArgs& A, int64_t idx, int32_t& t, int32_t& sc) {
    const int nch = 1 << A.s;
    const int64_t e = idx >> A.s;
    const int c = (int)(idx & (nch - 1));
    t = A.refine_src ? A.ftgt[e] : A.ftgt[e] * nch + c;
    sc = A.refine_src ? A.fsrc[e] * nch + c : A.fsrc[e];
}
__global__ void march_classify_k(MarchArgs A, uint8_t* codes) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (A.nfail << A.s)) return;
    int32_t t, sc;
    march_decode(A, idx, t, sc);
    const int64_t gt = A.off_t + t, gs = A.off_s + sc;
    uint8_t code = 0;
    if (A.box_count[gt] > 0 && A.count_s[gs] > 0) code = admissible2(A.ctr, A.rad, gt, A.ctr_s, A.rad_s, gs, A.theta) ? 1 : 2;
    codes[idx] = code;
}
__global__ void march_compact_k(MarchArgs A, const uint8_t* codes, const unsigned long long* S, int32_t* wtgt, int32_t* wsrc, int32_t* ftgt2,
                                int32_t* fsrc2) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (A.nfail << A.s)) return;
    int32_t t, sc;
    march_decode(A, idx, t, sc);
    const uint8_t c = codes[idx];
    const unsigned long long sv = S[idx];
    if (c == 1) {
        const int64_t o = (int64_t)(sv & 0xffffffffull);
        wtgt[o] = (int32_t)(A.off_t + t);
        wsrc[o] = (int32_t)(A.off_s + sc);
    } else if (c == 2) {
        const int64_t o = (int64_t)(sv >> 32);
        ftgt2[o] = t;
        fsrc2[o] = sc;
    }
}
__global__ void count_keys_k(const int32_t* keys, int64_t n, unsigned long long* cnt) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicAdd(cnt + keys[i], 1ull);
}
struct CntLoad {
    const unsigned long long* p;
    int64_t n;
    __device__ int64_t operator()(int64_t i) const { return i < n ? (int64_t)p[i] : 0; }
};

}  // namespace

void build_tree(Plan& P, const void* d_positions, cudaStream_t st) {
    if (P.dtype == FMM_F32) build_tree_t<float, uint32_t>(P, (const float*)d_positions, st);
    else build_tree_t<double, uint64_t>(P, (const double*)d_positions, st);
}

// after the strong list exists: number of P2P particle pairs and the P2P work items
static void finish_lists(Plan& P, cudaStream_t st) {
    const int L = P.L;
    DevBuf<unsigned long long> cnt;
    cnt.alloc(2);
    FMM_CUDA_CHECK(cudaMemsetAsync(cnt.p, 0, 16, st));
    const Plan& PS = P.S ? *P.S : P;  // hierarchy of the sources
    const int32_t* scnt = PS.box_count.p + PS.level_off[PS.L];
    P.strong_touch.alloc(P.n_strong);
    if (P.n_strong > 0) {
        const size_t to = (size_t)P.level_off[L] * 3, so = (size_t)PS.level_off[PS.L] * 3;
        if (P.dtype == FMM_F32)
            strong_touch_k<float><<<nblocks(P.n_leaves, 128), 128, 0, st>>>(P.strong_off.p, P.strong_src.p, (const float*)P.box_lo.p + to, (const float*)P.box_hi.p + to,
                                                                            (const float*)PS.box_lo.p + so, (const float*)PS.box_hi.p + so, P.n_leaves, P.strong_touch.p);
        else
            strong_touch_k<double><<<nblocks(P.n_leaves, 128), 128, 0, st>>>(P.strong_off.p, P.strong_src.p, (const double*)P.box_lo.p + to, (const double*)P.box_hi.p + to,
                                                                             (const double*)PS.box_lo.p + so, (const double*)PS.box_hi.p + so, P.n_leaves, P.strong_touch.p);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    count_p2p_k<<<nblocks(P.n_leaves, 256), 256, 0, st>>>(P.strong_off.p, P.strong_src.p, P.box_count.p + P.level_off[L], scnt, P.n_leaves, cnt.p);
    FMM_CUDA_CHECK(cudaGetLastError());
    unsigned long long h[2] = {0, 0};
    FMM_CUDA_CHECK(cudaMemcpyAsync(h, cnt.p, 16, cudaMemcpyDeviceToHost, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    P.n_p2p_pairs = (int64_t)h[0];
    P.p2p_src_total = (int64_t)h[1];
    build_p2p_items(P, st, P.deterministic);
    // coarsest level that holds a weak pair: above it no multipole is read and no local expansion is non-zero, so the M2M and
    // L2L passes stop there (one point set: sources sit on the target's level or one finer, PAPER.md:122-131 / reading S9)
    P.top_level = 0;
    if (!P.S && (int)P.weak_level_off.size() == L + 2) {
        int t = 0;
        while (t < L && P.weak_level_off[t + 1] == P.weak_level_off[t]) ++t;
        P.top_level = t;
    }
}

// Work items of the P2P kernels: the strong list of a target leaf cut into segments (p2p_segments_k).  single_segment: one item per
// leaf whatever its length -- no partial sums to combine with atomics (fmm_plan_set_deterministic).
void build_p2p_items(Plan& P, cudaStream_t st, bool single_segment) {
    const int L = P.L;
    const Plan& PS = P.S ? *P.S : P;
    const int32_t* scnt = PS.box_count.p + PS.level_off[PS.L];
    const unsigned long long h1 = (unsigned long long)P.p2p_src_total;
    {
        // work items of the P2P kernel: budget = twice the mean number of source particles per target leaf (at least 1024)
        const int32_t* lcnt = P.box_count.p + P.level_off[L];
        const int64_t mean_src = (int64_t)(h1 / (unsigned long long)(P.n_leaves > 0 ? P.n_leaves : 1));
        int64_t budget = mean_src * 2 > 1024 ? mean_src * 2 : 1024;
        // small problems: fewer target leaves than the chip has warp slots -- cut the lists finer (down to 64 source particles
        // per item; a list is cut between source leaves) so that about 16 warps per SM find work; the partial sums of a leaf are then
        // combined with atomics.  Config 1 (N = 4096, fp64, 64 leaves of 64): 8 warps per SM / 128 sources 43.0 us per evaluate, this 32.9 us
        const int64_t want_items = 148 * 16;
        if (P.n_leaves < want_items) {
            const int64_t fine = (int64_t)(h1 / (unsigned long long)want_items);
            budget = std::min(budget, std::max<int64_t>(64, fine));
        }
        if (single_segment) budget = INT64_MAX / 4;
        DevBuf<int32_t> nseg, any_multi;
        DevBuf<int64_t> seg_off, scratch;
        nseg.alloc(P.n_leaves);
        any_multi.alloc(1);
        FMM_CUDA_CHECK(cudaMemsetAsync(any_multi.p, 0, sizeof(int32_t), st));
        seg_off.alloc(P.n_leaves + 1);
        scratch.alloc(scan_scratch_elems(P.n_leaves + 1));
        p2p_segments_k<<<nblocks(P.n_leaves, 128), 128, 0, st>>>(P.strong_off.p, P.strong_src.p, P.box_start.p + P.level_off[L], lcnt, scnt, P.n_leaves, budget, nseg.p, nullptr, nullptr,
                                                                 any_multi.p);
        FMM_CUDA_CHECK(cudaGetLastError());
        exclusive_scan<int64_t>(SegLoad{nseg.p, P.n_leaves}, seg_off.p, P.n_leaves + 1, scratch.p, st);
        int64_t n_items = 0;
        int32_t multi = 0;
        FMM_CUDA_CHECK(cudaMemcpyAsync(&n_items, seg_off.p + P.n_leaves, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(&multi, any_multi.p, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        P.n_p2p_items = n_items;
        P.p2p_multi = multi != 0;
        P.p2p_item_off.alloc(P.n_leaves + 1);
        FMM_CUDA_CHECK(cudaMemcpyAsync(P.p2p_item_off.p, seg_off.p, (P.n_leaves + 1) * sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
        P.p2p_items.alloc((size_t)n_items * sizeof(P2PItem));
        if (n_items > 0) {
            p2p_segments_k<<<nblocks(P.n_leaves, 128), 128, 0, st>>>(P.strong_off.p, P.strong_src.p, P.box_start.p + P.level_off[L], lcnt, scnt, P.n_leaves, budget, nseg.p, seg_off.p,
                                                                     reinterpret_cast<P2PItem*>(P.p2p_items.p), nullptr);
            FMM_CUDA_CHECK(cudaGetLastError());
        }
    }
}

// stable LSD radix sort of (key, value) pairs by key in [0, n_keys) and the CSR offsets of the keys (n_keys + 1, device)
static void sort_by_key(DevBuf<int32_t>& keys, DevBuf<int32_t>& vals, int64_t n, int64_t n_keys, int64_t* off_out, cudaStream_t st) {
    DevBuf<unsigned long long> cnt;
    DevBuf<int64_t> scr64;
    cnt.alloc(n_keys + 1);
    scr64.alloc(scan_scratch_elems(n_keys + 1));
    FMM_CUDA_CHECK(cudaMemsetAsync(cnt.p, 0, (n_keys + 1) * sizeof(unsigned long long), st));
    if (n > 0) {
        int bits = 8;
        while (((int64_t)1 << bits) < n_keys) bits += 8;
        DevBuf<int32_t> kb, vb, hist, scr;
        kb.alloc(n); vb.alloc(n);
        const int nblk = (int)((n + RS_TILE - 1) / RS_TILE);
        hist.alloc((size_t)256 * nblk + 1);
        scr.alloc(scan_scratch_elems((int64_t)256 * nblk));
        const int where = radix_sort_pairs<uint32_t>(reinterpret_cast<uint32_t*>(keys.p), vals.p, reinterpret_cast<uint32_t*>(kb.p), vb.p, n, bits,
                                                     hist.p, scr.p, st);
        if (where == 1) {
            FMM_CUDA_CHECK(cudaMemcpyAsync(keys.p, kb.p, n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
            FMM_CUDA_CHECK(cudaMemcpyAsync(vals.p, vb.p, n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        }
        count_keys_k<<<nblocks(n, 256), 256, 0, st>>>(keys.p, n, cnt.p);
        FMM_CUDA_CHECK(cudaGetLastError());
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));  // temporaries are freed on scope exit
    }
    exclusive_scan<int64_t>(CntLoad{cnt.p, n_keys}, off_out, n_keys + 1, scr64.p, st);
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
}

// mean radius of the non-empty boxes of every level ("average box radius").  The oracle sums a level in box order in
// fp64; so does the device: one warp per level reads 32 radii at a time (coalesced) and lane 0 adds them one after the other with
// __dadd_rn, so the comparison of two levels takes the same decision on both sides bit for bit.  A dependent chain of n additions:
// 0.1 ms for the 32 768 leaves of N = 1M, N_max = 128.
__global__ void mean_radius_k(const double* __restrict__ rad, const int32_t* __restrict__ cnt, const int64_t* __restrict__ level_off, double* __restrict__ mean) {
    const int l = blockIdx.x, lane = threadIdx.x;
    const int64_t g0 = level_off[l], g1 = level_off[l + 1];
    double sum = 0.0;
    int64_t n = 0;
    for (int64_t g = g0; g < g1; g += 32) {
        const bool in = g + lane < g1;
        const double r = in ? rad[g + lane] : 0.0;
        const bool use = in && cnt[g + lane] > 0;
        const unsigned m = __ballot_sync(0xffffffffu, use);
        n += __popc(m);
        if (m == 0xffffffffu) {
#pragma unroll
            for (int k = 0; k < 32; ++k) sum = __dadd_rn(sum, __shfl_sync(0xffffffffu, r, k));
        } else {
            for (int k = 0; k < 32; ++k) {
                const double rk = __shfl_sync(0xffffffffu, r, k);
                if ((m >> k) & 1u) sum = __dadd_rn(sum, rk);
            }
        }
    }
    if (lane == 0) mean[l] = n ? __ddiv_rn(sum, (double)n) : 0.0;
}

static std::vector<double> mean_radii(const Plan& P, cudaStream_t st) {
    DevBuf<int64_t> off;
    DevBuf<double> mean;
    off.alloc(P.L + 2);
    mean.alloc(P.L + 1);
    FMM_CUDA_CHECK(cudaMemcpyAsync(off.p, P.level_off.data(), (P.L + 2) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    mean_radius_k<<<P.L + 1, 32, 0, st>>>(P.box_rad.p, P.box_count.p, off.p, mean.p);
    FMM_CUDA_CHECK(cudaGetLastError());
    std::vector<double> m(P.L + 1, 0.0);
    FMM_CUDA_CHECK(cudaMemcpyAsync(m.data(), mean.p, (P.L + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    return m;  // L + 1 numbers: the host only compares them to pick the next launch of the march
}

// Level marching over the target hierarchy (P) and the source hierarchy (P.S, or P itself when sources and targets share one
// hierarchy).  One hierarchy: the fixed sequence of reading S9.  Two hierarchies: PAPER.md:85-88 -- refine the side with the
// larger mean box radius, ties -> sources, an exhausted side -> the other.
static void build_lists_cross(Plan& P, cudaStream_t st) {
    const Plan& PS = P.S ? *P.S : P;
    const int s = P.s, L = P.L, Lsrc = PS.L;
    const int nch = 1 << s;
    std::vector<double> mr_t, mr_s;
    if (P.S) { mr_t = mean_radii(P, st); mr_s = mean_radii(PS, st); }
    P.weak_off.alloc(P.n_boxes + 1);
    P.weak_level_off.assign(L + 2, 0);
    DevBuf<int32_t> ftgt, fsrc;
    ftgt.alloc(1); fsrc.alloc(1);
    FMM_CUDA_CHECK(cudaMemsetAsync(ftgt.p, 0, 4, st));  // (root, root) is the first candidate pair
    FMM_CUDA_CHECK(cudaMemsetAsync(fsrc.p, 0, 4, st));
    int64_t nfail = 1;
    std::vector<DevBuf<int32_t>> wt(L + Lsrc + 2), ws(L + Lsrc + 2);
    std::vector<int64_t> wn(L + Lsrc + 2, 0);
    int lt = 0, ls = 0, step = 0;
    int64_t n_weak = 0;
    P.march_steps.assign({0, 0});
    if (P.S) {
        // the root pair itself may already be admissible when the two point sets are far apart: classify it like any other
        // candidate by starting the march one step "before" the roots: a single candidate (0, 0) at (lt, ls) = (0, 0)
        MarchArgs A{ftgt.p, fsrc.p, 1, 0, 1, 0, 0, P.box_count.p, P.box_ctr.p, P.box_rad.p, PS.box_count.p, PS.box_ctr.p, PS.box_rad.p, P.theta};
        DevBuf<uint8_t> code0;
        code0.alloc(1);
        march_classify_k<<<1, 32, 0, st>>>(A, code0.p);
        FMM_CUDA_CHECK(cudaGetLastError());
        uint8_t h = 0;
        FMM_CUDA_CHECK(cudaMemcpyAsync(&h, code0.p, 1, cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        if (h == 1) {  // one weak pair (root, root); nothing fails
            wt[step].alloc(1); ws[step].alloc(1); wn[step] = 1;
            FMM_CUDA_CHECK(cudaMemsetAsync(wt[step].p, 0, 4, st));
            FMM_CUDA_CHECK(cudaMemsetAsync(ws[step].p, 0, 4, st));
            n_weak = 1;
            nfail = 0;
        }
        ++step;
    }
    while (!(lt == L && ls == Lsrc)) {
        int refine_src;
        if (!P.S) refine_src = lt == ls;  // PAPER.md:85-87 for one hierarchy: sources first, then targets
        else if (ls == Lsrc) refine_src = 0;
        else if (lt == L) refine_src = 1;
        else refine_src = !(mr_t[lt] > mr_s[ls]);
        if (refine_src) ++ls; else ++lt;
        P.march_steps.push_back(lt); P.march_steps.push_back(ls);
        const int64_t total = nfail << s;
        MarchArgs A{ftgt.p, fsrc.p, nfail, s, refine_src, P.level_off[lt], PS.level_off[ls], P.box_count.p, P.box_ctr.p, P.box_rad.p,
                    PS.box_count.p, PS.box_ctr.p, PS.box_rad.p, P.theta};
        DevBuf<uint8_t> codes;
        DevBuf<unsigned long long> S, scr;
        codes.alloc(total + 1);
        S.alloc(total + 1);
        scr.alloc(scan_scratch_elems(total + 1));
        if (total > 0) {
            march_classify_k<<<nblocks(total, 256), 256, 0, st>>>(A, codes.p);
            FMM_CUDA_CHECK(cudaGetLastError());
        }
        exclusive_scan<unsigned long long, CodeLoad>(CodeLoad{codes.p, total}, S.p, total + 1, scr.p, st);
        unsigned long long tot = 0;
        FMM_CUDA_CHECK(cudaMemcpyAsync(&tot, S.p + total, sizeof(tot), cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        const int64_t nweak_l = (int64_t)(tot & 0xffffffffull), nfail2 = (int64_t)(tot >> 32);
        if (nweak_l >= 0xffffffffll || nfail2 >= 0xffffffffll) {
            set_error("interaction list of one step exceeds 2^32-1 pairs");
            throw CudaFail{FMM_ERR_UNSUPPORTED};
        }
        wt[step].alloc(nweak_l); ws[step].alloc(nweak_l); wn[step] = nweak_l;
        DevBuf<int32_t> ftgt2, fsrc2;
        ftgt2.alloc(nfail2); fsrc2.alloc(nfail2);
        if (total > 0) {
            march_compact_k<<<nblocks(total, 256), 256, 0, st>>>(A, codes.p, S.p, wt[step].p, ws[step].p, ftgt2.p, fsrc2.p);
            FMM_CUDA_CHECK(cudaGetLastError());
        }
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        std::swap(ftgt.p, ftgt2.p); std::swap(ftgt.n, ftgt2.n);
        std::swap(fsrc.p, fsrc2.p); std::swap(fsrc.n, fsrc2.n);
        nfail = nfail2;
        n_weak += nweak_l;
        ++step;
    }
    (void)nch;
    if (n_weak > 0x7fffff00ll || nfail > 0x7fffff00ll) { set_error("interaction lists exceed 2^31 pairs"); throw CudaFail{FMM_ERR_UNSUPPORTED}; }

    P.n_weak = n_weak;
    P.weak_tgt.alloc(n_weak); P.weak_src.alloc(n_weak);
    {
        int64_t o = 0;
        for (int k = 0; k < step; ++k) {
            if (!wn[k]) continue;
            FMM_CUDA_CHECK(cudaMemcpyAsync(P.weak_tgt.p + o, wt[k].p, wn[k] * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
            FMM_CUDA_CHECK(cudaMemcpyAsync(P.weak_src.p + o, ws[k].p, wn[k] * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
            o += wn[k];
        }
    }
    sort_by_key(P.weak_tgt, P.weak_src, n_weak, P.n_boxes, P.weak_off.p, st);
    for (int l = 0; l <= L + 1; ++l)  // weak pairs are sorted by target id, hence by target level
        FMM_CUDA_CHECK(cudaMemcpyAsync(&P.weak_level_off[l], P.weak_off.p + P.level_off[l], sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    // strong list = pairs still failing at (L, L) (rule L3)
    P.n_strong = nfail;
    P.strong_off.alloc(P.n_leaves + 1);
    P.strong_src.alloc(nfail);
    sort_by_key(ftgt, fsrc, nfail, P.n_leaves, P.strong_off.p, st);
    FMM_CUDA_CHECK(cudaMemcpyAsync(P.strong_src.p, fsrc.p, nfail * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
}

void build_lists(Plan& P, cudaStream_t st) {
    cudaEvent_t e0, e1;
    FMM_CUDA_CHECK(cudaEventCreate(&e0));
    FMM_CUDA_CHECK(cudaEventCreate(&e1));
    FMM_CUDA_CHECK(cudaEventRecord(e0, st));
    const int s = P.s, L = P.L;
    if (P.cross_level) {
        build_lists_cross(P, st);
        finish_lists(P, st);
        FMM_CUDA_CHECK(cudaEventRecord(e1, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        float msx = 0;
        cudaEventElapsedTime(&msx, e0, e1);
        P.plan_ms[2] = msx;
        cudaEventDestroy(e0); cudaEventDestroy(e1);
        return;
    }
    P.weak_off.alloc(P.n_boxes + 1);
    FMM_CUDA_CHECK(cudaMemsetAsync(P.weak_off.p, 0, (P.n_boxes + 1) * sizeof(int64_t), st));
    P.weak_level_off.assign(L + 2, 0);

    // level 0: the pair (root, root) always fails eq. (4) (d = 0)
    DevBuf<int32_t> ftgt, fsrc;
    DevBuf<int64_t> foff;
    ftgt.alloc(1); fsrc.alloc(1); foff.alloc(2);
    {
        const int32_t z = 0;
        const int64_t o[2] = {0, 1};
        FMM_CUDA_CHECK(cudaMemcpyAsync(ftgt.p, &z, 4, cudaMemcpyHostToDevice, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(fsrc.p, &z, 4, cudaMemcpyHostToDevice, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(foff.p, o, 16, cudaMemcpyHostToDevice, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    }
    int64_t nfail = 1;
    std::vector<DevBuf<int32_t>> wt(L + 1), ws(L + 1);
    std::vector<int64_t> wn(L + 1, 0);
    int64_t weak_base = 0;
    for (int l = 1; l <= L; ++l) {
        const int64_t nb_child = (int64_t)1 << (s * l);
        const int64_t total = nfail << (2 * s);
        ExpandArgs A{ftgt.p, fsrc.p, foff.p, nfail, s, P.level_off[l], P.box_count.p, P.box_ctr.p, P.box_rad.p, P.theta};
        DevBuf<uint8_t> codes;
        DevBuf<unsigned long long> S, scr;
        codes.alloc(total + 1);
        S.alloc(total + 1);
        scr.alloc(scan_scratch_elems(total + 1));
        if (total > 0) {
            expand_classify_k<<<nblocks(total, 256), 256, 0, st>>>(A, codes.p);
            FMM_CUDA_CHECK(cudaGetLastError());
        }
        exclusive_scan<unsigned long long, CodeLoad>(CodeLoad{codes.p, total}, S.p, total + 1, scr.p, st);
        unsigned long long tot = 0;
        FMM_CUDA_CHECK(cudaMemcpyAsync(&tot, S.p + total, sizeof(tot), cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        const int64_t nweak_l = (int64_t)(tot & 0xffffffffull), nfail2 = (int64_t)(tot >> 32);
        if (nweak_l >= 0xffffffffll || nfail2 >= 0xffffffffll) {
            set_error("interaction list of one level exceeds 2^32-1 pairs");
            throw CudaFail{FMM_ERR_UNSUPPORTED};
        }
        wt[l].alloc(nweak_l); ws[l].alloc(nweak_l); wn[l] = nweak_l;
        DevBuf<int32_t> ftgt2, fsrc2;
        DevBuf<int64_t> foff2;
        ftgt2.alloc(nfail2); fsrc2.alloc(nfail2); foff2.alloc(nb_child + 1);
        if (total > 0) {
            expand_compact_k<<<nblocks(total, 256), 256, 0, st>>>(A, codes.p, S.p, wt[l].p, ws[l].p, ftgt2.p, fsrc2.p);
            FMM_CUDA_CHECK(cudaGetLastError());
        }
        expand_offsets_k<<<nblocks(nb_child + 1, 256), 256, 0, st>>>(A, S.p, nb_child, total, weak_base, P.weak_off.p, foff2.p);
        FMM_CUDA_CHECK(cudaGetLastError());
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        weak_base += nweak_l;
        P.weak_level_off[l + 1] = weak_base;
        std::swap(ftgt.p, ftgt2.p); std::swap(ftgt.n, ftgt2.n);
        std::swap(fsrc.p, fsrc2.p); std::swap(fsrc.n, fsrc2.n);
        std::swap(foff.p, foff2.p); std::swap(foff.n, foff2.n);
        nfail = nfail2;
    }
    // the expand_offsets kernel wrote weak_off[off_l + t] for t = 0..nb_l (the entry t = nb_l is the next level's first row
    // or the final end); level 0 rows are zero.  Make sure the final end is set when L == 0.
    P.n_weak = weak_base;
    if (L == 0) P.weak_level_off[1] = 0;
    {
        const int64_t endv = weak_base;
        FMM_CUDA_CHECK(cudaMemcpyAsync(P.weak_off.p + P.n_boxes, &endv, sizeof(int64_t), cudaMemcpyHostToDevice, st));
    }
    P.weak_src.alloc(P.n_weak); P.weak_tgt.alloc(P.n_weak);
    for (int l = 1; l <= L; ++l) {
        if (!wn[l]) continue;
        FMM_CUDA_CHECK(cudaMemcpyAsync(P.weak_tgt.p + P.weak_level_off[l], wt[l].p, wn[l] * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(P.weak_src.p + P.weak_level_off[l], ws[l].p, wn[l] * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    }
    // strong list = failing pairs of the leaf level (rule L3), already CSR by target leaf
    P.n_strong = nfail;
    P.strong_off.alloc(P.n_leaves + 1);
    P.strong_src.alloc(nfail);
    FMM_CUDA_CHECK(cudaMemcpyAsync(P.strong_off.p, foff.p, (P.n_leaves + 1) * sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
    FMM_CUDA_CHECK(cudaMemcpyAsync(P.strong_src.p, fsrc.p, nfail * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    finish_lists(P, st);
    FMM_CUDA_CHECK(cudaEventRecord(e1, st));
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    P.plan_ms[2] = ms;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
}


// ---------------------------------------------------------------------------------------------- adjoint view
// The transposed evaluate runs the forward kernels on a VIEW of the plan with the roles of sources and targets exchanged: the view's
// target hierarchy is the plan's source hierarchy and vice versa (all hierarchy arrays are aliases, nothing is copied), and its
// interaction lists are the plan's lists transposed: weak pairs sorted by (source, target), strong list CSR by source leaf.
namespace {
__global__ void expand_rows_k(const int64_t* off, int64_t n_rows, int32_t* row_of) {  // CSR offsets -> row index per entry (warp per row)
    const int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (r >= n_rows) return;
    for (int64_t e = off[r] + (threadIdx.x & 31); e < off[r + 1]; e += 32) row_of[e] = (int32_t)r;
}

void alias_hierarchy(Plan& V, const Plan& H) {
    V.device = H.device;
    V.N = H.N; V.p = H.p; V.N_max = H.N_max; V.s = H.s; V.L = H.L; V.dtype = H.dtype; V.theta = H.theta;
    V.K = H.K; V.Kp = H.Kp; V.n_boxes = H.n_boxes; V.n_leaves = H.n_leaves; V.level_off = H.level_off; V.max_leaf = H.max_leaf;
    V.perm.alias(H.perm); V.pos_tree.alias(H.pos_tree); V.box_start.alias(H.box_start); V.box_count.alias(H.box_count);
    V.box_lo.alias(H.box_lo); V.box_hi.alias(H.box_hi); V.box_ctr.alias(H.box_ctr); V.box_rad.alias(H.box_rad); V.box_scale.alias(H.box_scale);
    V.srcg.alias(H.srcg); V.src_slot.alias(H.src_slot); V.src_G = H.src_G;
    V.pq.alias(H.pq);
}
}  // namespace

void build_adjoint_view(Plan& P, cudaStream_t st) {
    if (P.adj) return;
    const Plan& HS = P.S ? *P.S : P;  // hierarchy of the plan's sources = the view's targets
    std::unique_ptr<Plan> Vp(new Plan());
    Plan& V = *Vp;
    alias_hierarchy(V, HS);
    V.cross_level = 1;
    V.no_split = true;  // a transposed weak pair may join a target with a COARSER source: the whole upward pass must precede the M2L
    V.m2l_variant = P.m2l_variant;
    if (P.S) {
        V.S.reset(new Plan());
        alias_hierarchy(*V.S, P);
        V.S->Mc.alias(P.Lc);   // multipoles of the view's sources live on the plan's target hierarchy: its local array is free
        V.Lc.alias(P.S->Mc);   // and the other way round
    } else {
        V.Mc.alias(P.Lc);
        V.Lc.alias(P.Mc);
    }
    const size_t es = P.dtype == FMM_F32 ? 4 : 8;
    V.near.alloc((size_t)V.N * 4 * es);
    // weak list: (target, source) pairs of the plan -> keys = source, values = target; the plan's order (target, source) and a
    // stable sort by source give the canonical order (source, target) of the view
    V.n_weak = P.n_weak;
    V.weak_tgt.alloc(P.n_weak); V.weak_src.alloc(P.n_weak);
    V.weak_off.alloc(V.n_boxes + 1);
    if (P.n_weak > 0) {
        FMM_CUDA_CHECK(cudaMemcpyAsync(V.weak_tgt.p, P.weak_src.p, P.n_weak * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        FMM_CUDA_CHECK(cudaMemcpyAsync(V.weak_src.p, P.weak_tgt.p, P.n_weak * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    }
    sort_by_key(V.weak_tgt, V.weak_src, P.n_weak, V.n_boxes, V.weak_off.p, st);
    // strong list: CSR by target leaf -> (target leaf, source leaf) pairs -> CSR by source leaf
    V.n_strong = P.n_strong;
    DevBuf<int32_t> keys, vals;
    keys.alloc(P.n_strong); vals.alloc(P.n_strong);
    V.strong_off.alloc(V.n_leaves + 1);
    V.strong_src.alloc(P.n_strong);
    if (P.n_strong > 0) {
        FMM_CUDA_CHECK(cudaMemcpyAsync(keys.p, P.strong_src.p, P.n_strong * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        expand_rows_k<<<nblocks(P.n_leaves * 32, 256), 256, 0, st>>>(P.strong_off.p, P.n_leaves, vals.p);
        FMM_CUDA_CHECK(cudaGetLastError());
    }
    sort_by_key(keys, vals, P.n_strong, V.n_leaves, V.strong_off.p, st);
    if (P.n_strong > 0) FMM_CUDA_CHECK(cudaMemcpyAsync(V.strong_src.p, vals.p, P.n_strong * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    finish_lists(V, st);
    if (m2l_geo_wanted(V.p, V.dtype) && V.n_weak > 0) m2l_geo_prepare(V, st);
    FMM_CUDA_CHECK(cudaStreamSynchronize(st));
    P.adj = std::move(Vp);
}

}  // namespace fmm
