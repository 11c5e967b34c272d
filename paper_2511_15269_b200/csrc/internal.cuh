// internal.cuh -- shared declarations of the CUDA path (plan struct, error helpers, device tables).
// Not part of the public boundary (include/fmm.h) and not shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <memory>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/fmm.h"

namespace fmm {

constexpr int PMAX = FMM_P_MAX;
constexpr int KMAX = (PMAX + 1) * (PMAX + 1);

void set_error(const std::string& msg);

struct CudaFail {
    fmm_status st;
};

#define FMM_CUDA_CHECK(expr)                                                                               \
    do {                                                                                                   \
        cudaError_t _e = (expr);                                                                           \
        if (_e != cudaSuccess) {                                                                           \
            ::fmm::set_error(std::string(#expr) + ": " + cudaGetErrorString(_e));                          \
            throw ::fmm::CudaFail{_e == cudaErrorMemoryAllocation ? FMM_ERR_ALLOC : FMM_ERR_CUDA};         \
        }                                                                                                  \
    } while (0)

// Device memory comes from the device's stream-ordered pool (cudaMallocAsync / cudaFreeAsync on the stream of the API call
// that is running, see AllocScope): the many short-lived scratch buffers of a plan build are recycled inside the pool
// instead of going through cudaMalloc / cudaFree (each of which synchronises the device), and a later plan of similar
// size finds its memory already mapped.  Every API call that allocates ends with a stream synchronisation, so plan
// buffers are safe to use from any stream afterwards.
inline cudaStream_t& alloc_stream() {
    static thread_local cudaStream_t s = nullptr;
    return s;
}
struct AllocScope {
    cudaStream_t prev;
    explicit AllocScope(cudaStream_t st) : prev(alloc_stream()) { alloc_stream() = st; }
    ~AllocScope() { alloc_stream() = prev; }
};

// device buffer owned by the plan
template <typename T>
struct DevBuf {
    T* p = nullptr;
    size_t n = 0;
    bool owned = true;  // false: an alias of another buffer (adjoint view of a plan); never freed here
    void alloc(size_t count) {
        release();
        n = count;
        if (count) FMM_CUDA_CHECK(cudaMallocAsync((void**)&p, count * sizeof(T), alloc_stream()));
    }
    void alias(const DevBuf& o) {
        release();
        p = o.p;
        n = o.n;
        owned = false;
    }
    void release() {
        if (p && owned) cudaFreeAsync(p, alloc_stream());
        p = nullptr;
        n = 0;
        owned = true;
    }
    ~DevBuf() { release(); }
    DevBuf() = default;
    DevBuf(const DevBuf&) = delete;
    DevBuf& operator=(const DevBuf&) = delete;
};

// Constant tables of the normalised operators (built once per DEVICE, host fp64 -> device):
//   Bmat : per degree n a (2n+1)x(2n+1) row-major block at offset boff(n) = n(2n-1)(2n+1)/3;
//          polar rotation Q_n(theta) = B_n Z_n(theta) B_n^T  (exact identity, B_n derived from d^n(pi/2))
//   Hm2l : H[m][n][k] = (n+k)! / sqrt((n-m)!(n+m)!(k-m)!(k+m)!) * (-1)^(k+m)      (M2L z-shift weights)
//   Am2m : A[m][n][k] = sqrt((n-m)!(n+m)!/((k-m)!(k+m)!)) / (n-k)!   for k<=n      (M2M; L2L uses A[m][k][n])
//   gnorm: g[idx(n,m)] = sqrt((n-|m|)!(n+|m|)!) * (m ? sqrt2 : 1)
struct Tables {
    double* d_B = nullptr;   // sum_n (2n+1)^2 doubles
    float* d_Bf = nullptr;   // same in fp32
    double* d_H = nullptr;   // (PMAX+1)^3
    double* d_A = nullptr;   // (PMAX+1)^3
    double* d_g = nullptr;   // KMAX
    std::vector<double> h_B; // host copy (used by the unrolled-kernel self check)
};
// Everything the library sets up once per device lives here (tables.cu): operator tables, the __constant__ copies of g_n^m,
// the memory-pool threshold.  One process may hold plans on several devices; a plan remembers its device (Plan::device) and
// every entry point checks that it is the current one.  Creation and the one-time steps are guarded by mutexes, so plans on
// different devices may be created and used from different host threads.
constexpr int MAX_DEVICES = 64;
struct DeviceCtx {
    int dev = -1;
    Tables tab;
    std::mutex mu;                // guards the lazy steps below
    bool const_uploaded = false;  // evaluate.cu: c_g / c_gf
    bool pool_ready = false;      // api.cu: release threshold of the default memory pool
};
DeviceCtx& device_ctx(int dev);   // throws CudaFail; builds and uploads the tables on first use (dev must be the current device)
int current_device();             // cudaGetDevice or throws
inline const Tables& tables(int dev) { return device_ctx(dev).tab; }

// one-time, per-device cudaFuncSetAttribute of a kernel instantiation: `static AttrOnce once; once.ensure(dev, [&]{...});`
struct AttrOnce {
    std::atomic<unsigned long long> mask{0};
    template <class F>
    void ensure(int dev, F&& f) {
        const unsigned long long bit = 1ull << (dev & (MAX_DEVICES - 1));
        if (mask.load(std::memory_order_acquire) & bit) return;
        f();  // idempotent: two threads racing here both set the same attribute
        mask.fetch_or(bit, std::memory_order_release);
    }
};
__host__ __device__ inline int boff(int n) { return n * (2 * n - 1) * (2 * n + 1) / 3; }

// P2P work item (plan.cu p2p_segments_k, p2p_fast.cu): one segment of the strong list of a target leaf
struct P2PItem {
    int32_t start, cnt;  // particle range of the target leaf (tree order)
    int64_t e0, e1;      // entries [e0, e1) of strong_src; e1 < 0 encodes ~e1 and "the leaf has several segments": partial
                         // sums are then combined with atomics
};

struct Plan {
    int device = 0;  // the CUDA device the plan's memory lives on
    int64_t N = 0;
    int p = 0, N_max = 0, s = 0, L = 0;
    fmm_dtype dtype = FMM_F32;
    double theta = 0.77;
    int cross_level = 0;  // 1: level-marching lists
    int K = 0, Kp = 0;  // (p+1)^2 and the padded row stride of coefficient arrays
    int64_t n_boxes = 0, n_leaves = 0, n_weak = 0, n_strong = 0, n_p2p_pairs = 0;
    std::vector<int64_t> level_off;  // L+2
    std::vector<int64_t> weak_level_off;  // L+2: offsets of each level's pairs in the weak list
    int m2l_variant = 0;
    int max_leaf = 0;  // largest leaf population
    // Separate sources and targets (fmm_plan_create_targets): THIS plan holds the hierarchy of the targets,
    // the local coefficients Lc, `near` and both lists (weak: target box id here -> source box id in S; strong: target leaf ->
    // source leaf of S); S holds the hierarchy of the sources, their permuted particles (pq, srcg) and the multipoles Mc.
    std::unique_ptr<Plan> S;
    // Adjoint evaluate (fmm_evaluate_adjoint): a view of this plan with the roles of sources and targets exchanged --
    // aliases of the hierarchy arrays plus the transposed interaction lists -- built on first use (plan.cu build_adjoint_view).
    // Declared after S: it is destroyed first, while the buffers it aliases are still alive.
    std::unique_ptr<Plan> adj;
    // Target-sharded evaluate (fmm_evaluate_shard_*): what shard `shard` of `n_shards` owns -- a contiguous range of target leaves,
    // i.e. a set of subtrees (the tree order is a Z-order), the weak pairs whose target is one of its boxes or one of
    // their ancestors (per level a contiguous piece of the list, which is sorted by target) and its P2P work items.  Host copy of the
    // few offsets involved, cached for the shard used last.
    struct Shard {
        int n_shards = 0, shard = -1;
        int64_t leaf_lo = 0, leaf_hi = 0;
        std::vector<int64_t> box_lo, box_hi;  // per level: level-local box range
        std::vector<int64_t> e0, e1;          // per level: weak pairs [e0, e1)
        int64_t item0 = 0, item1 = 0;         // P2P work items
    };
    mutable Shard shard_cache;
    int top_level = 0;      // M2M / L2L passes run between the leaf level and this one (finish_lists)
    bool no_split = false;  // evaluate schedule: never run the leaf-level M2L beside the M2M pass (sources may be coarser than targets)
    std::vector<int> march_steps;  // (l_trg, l_src) pairs visited by the level march (cross_level = 1 or separate targets)

    DevBuf<int32_t> perm;                 // N: tree order -> input index
    DevBuf<char> pos_tree;                // N x 3 dtype, tree order
    DevBuf<int32_t> box_start, box_count; // n_boxes
    DevBuf<char> box_lo, box_hi;          // n_boxes x 3 dtype
    DevBuf<double> box_ctr, box_rad;      // n_boxes x 3, n_boxes  (fp64 always)
    DevBuf<char> box_scale;               // n_boxes dtype: expansion length scale a_box
    DevBuf<int64_t> weak_off;             // n_boxes+1
    DevBuf<int32_t> weak_src, weak_tgt;   // n_weak (global ids)
    DevBuf<int64_t> strong_off;           // n_leaves+1
    DevBuf<int32_t> strong_src;           // n_strong (leaf indices)
    DevBuf<uint8_t> strong_touch;         // n_strong: 1 if the tight boxes of target and source leaf touch or overlap, i.e. a zero
                                          // distance is possible (the leaf itself; leaves sharing duplicated points): only those need the S3 mask
    // evaluate scratch
    DevBuf<char> pq;      // N x 4 dtype: (x,y,z,q) tree order
    DevBuf<char> Mc, Lc;  // n_boxes x Kp dtype: multipole / local coefficients (normalised, scaled)
    DevBuf<char> near;    // N x 4 dtype: (phi_near, grad phi_near) tree order, P2P -> L2P (which finalizes)
    mutable DevBuf<char> dip;  // N x 4 dtype: dipole moments of the sources in tree order (adjoint of the field), allocated on first use
    // fp32 P2P source groups (p2p_fast.cu): per leaf src_G groups of (-x[4], -y[4], -z[4], q[4]); src_slot[k] = 4*group + (i & 3)
    DevBuf<float> m2l_geo;   // xlate_fast.cu: per batch of 32 weak pairs a 1 KB geometry record (fp32, p <= 8)
    int64_t m2l_seg_e0[2] = {0, 0}, m2l_seg_rec[2] = {0, 0};  // the two segments of the weak list the records are batched by: first pair, first record
    DevBuf<char> p2p_items;  // n_p2p_items x P2PItem
    DevBuf<int64_t> p2p_item_off;  // n_leaves + 1: first work item of every target leaf (items are stored in leaf order)
    int64_t n_p2p_items = 0;
    int64_t p2p_src_total = 0;  // sum over the non-empty target leaves of the source particles in their strong lists
    bool p2p_multi = false;  // some leaf has more than one item: `near` is zeroed before P2P and those leaves use atomics
    DevBuf<float> srcg;
    DevBuf<int32_t> src_slot;
    int src_G = 0;
    DevBuf<char> h2d_q, d2h_out;  // staging for fmm_evaluate_host
    // fmm_evaluate_host_submit / _wait (api.cu): two calls may be in flight; the copies of one run on s_h2d / s_d2h beside the
    // evaluate of the other.  head = oldest call not yet waited for.
    struct HostSlot {
        DevBuf<char> q, out;
        cudaEvent_t e_in = nullptr, e_eval = nullptr, e_out = nullptr;
    };
    HostSlot hslot[2];
    int hs_head = 0, hs_count = 0;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    // internal streams / events of the concurrent evaluate schedule (evaluate.cu), created on first use
    mutable cudaStream_t s_far = nullptr, s_up = nullptr, s_near = nullptr;
    mutable cudaEvent_t e_fork = nullptr, e_perm = nullptr, e_p2m = nullptr, e_up = nullptr, e_near = nullptr, e_done = nullptr;
    // CUDA graphs of the evaluate schedule (evaluate.cu run_evaluate): the launches of one evaluate -- kernels, memsets and the
    // fork / join edges between the internal streams -- are captured once per set of caller pointers on s_cap and replayed with one
    // cudaGraphLaunch; a small cache because forward and adjoint evaluates alternate in an optimisation loop.
    struct EvalGraph {
        cudaGraphExec_t exec = nullptr;
        const void *q = nullptr, *dip = nullptr;
        void *pot = nullptr, *fld = nullptr;
        uint64_t stamp = ~0ull;  // Plan::epoch and the schedule switches the graph was captured under
        int seen = 0;            // evaluates with this key so far (the first runs plainly: one-time attribute / allocation work)
    };
    static constexpr int N_GRAPHS = 4;
    mutable EvalGraph graphs[N_GRAPHS];
    mutable int graph_next = 0;
    mutable cudaStream_t s_cap = nullptr;
    mutable int use_graph = 2;      // fmm_plan_set_graph: 0 never, 1 always, 2 (default) plans with fewer than 2^19 points; set to 0 if a capture fails
    uint64_t epoch = 0;             // bumped whenever arrays the graphs point into are rebuilt (update, deterministic switch)
    bool serial = false;  // true: every kernel on the caller's stream (fmm_plan_set_schedule)
    bool deterministic = false;  // fmm_plan_set_deterministic: serial schedule, no floating-point atomics with more than one contributor
    ~Plan() {
        for (EvalGraph& g : graphs)
            if (g.exec) cudaGraphExecDestroy(g.exec);
        for (HostSlot& h : hslot) {
            if (h.e_out && hs_count > 0) cudaEventSynchronize(h.e_out);
            for (cudaEvent_t e : {h.e_in, h.e_eval, h.e_out})
                if (e) cudaEventDestroy(e);
        }
        for (cudaStream_t q : {s_far, s_up, s_near, s_cap, s_h2d, s_d2h})
            if (q) cudaStreamDestroy(q);
        for (cudaEvent_t e : {e_fork, e_perm, e_p2m, e_up, e_near, e_done})
            if (e) cudaEventDestroy(e);
    }
    Plan() = default;
    double plan_ms[4] = {0, 0, 0, 0};
    double stage_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

// plan.cu
void build_tree(Plan& P, const void* d_positions, cudaStream_t st);
void build_lists(Plan& P, cudaStream_t st);
void build_p2p_items(Plan& P, cudaStream_t st, bool single_segment);  // (re)builds Plan::p2p_items; synchronises the stream
void build_adjoint_view(Plan& P, cudaStream_t st);  // fills P.adj (transposed lists; synchronises the stream)
// evaluate.cu
// d_q: charges (may be null = zero charges), d_dip: optional dipole moments (N_sources x 3, input order): the sources then also
// carry the potential -d . grad_source(1/|x - y|) (the transposed field operator of fmm_evaluate_adjoint); potential only
void run_evaluate(const Plan& P, const void* d_q, void* d_pot, void* d_field, cudaStream_t st, cudaEvent_t* ev /*8 or null*/, const void* d_dip = nullptr);
int64_t evaluate_launches(const Plan& P);  // kernels launched by one run_evaluate
// xlate_fast.cu: register kernels (one thread per translation).  kind 0 = M2M into level-1 from `level`, 1 = M2L (all
// levels, `level` ignored), 2 = L2L from level-1 into `level`.  Results are ADDED (atomically) to the output rows.
bool xlate_fast_available(int p, fmm_dtype dt);  // false if no register kernel exists for (p, dtype)
void xlate_work(int p, fmm_dtype dt, int kind, int64_t w[3]);  // {FMA, MUL, ADD} instructions of one translation (0 if generic only)
// kind 1: weak pairs [e0, e1); kinds 0 / 2: children [e0, e1) of `level` (level-local indices; e1 < 0: all)
void xlate_fast_launch(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0 = 0, int64_t e1 = -1);
// xlate_smem.cu: the same three operators for 9 <= p <= 12, one thread per translation with the state vector in shared memory
bool xlate_smem_available(int p, fmm_dtype dt);
void xlate_smem_launch(const Plan& P, int kind, int level, cudaStream_t st, int64_t e0, int64_t e1);
bool m2l_row_available(int p, fmm_dtype dt);     // deterministic M2L, one warp per target box (p <= 8)
void m2l_row_launch(const Plan& P, cudaStream_t st);
bool m2l_geo_wanted(int p, fmm_dtype dt);        // fp32, p <= 8: the M2L kernel reads per-pair geometry records
void m2l_geo_prepare(Plan& P, cudaStream_t st);  // plan time, after build_lists: writes Plan::m2l_geo
// p2p_fast.cu: fp32 near field + finalize, one target leaf per warp, packed f32x2 arithmetic
// want_field = false: potential only (cheaper inner loop); work items [item0, item1) of Plan::p2p_items (item1 < 0: all)
void p2p_fast_launch(const Plan& P, cudaStream_t st, bool want_field, int64_t item0 = 0, int64_t item1 = -1);
void p2p_fast64_launch(const Plan& P, cudaStream_t st, bool want_field, int64_t item0 = 0, int64_t item1 = -1);  // fp64: same mapping, scalar DFMA arithmetic
// evaluate.cu: target-sharded evaluate (see Plan::Shard); both run serially on st
void shard_box_range(int L, int s, int n_shards, int shard, int level, int64_t* b0, int64_t* b1);
void run_shard_upward(const Plan& P, int n_shards, int shard, const void* d_q, cudaStream_t st);
void run_shard_downward(const Plan& P, int n_shards, int shard, void* d_pot, void* d_field, cudaStream_t st);
// leaf multipoles of all leaves into the caller's rows, permuted particles in static device memory (fmm_leaf_multipoles_noalloc)
int64_t noalloc_max_particles(fmm_dtype dt);
void run_leaf_multipoles_noalloc(const Plan& P, const void* d_q, void* d_rows, cudaStream_t st);

}  // namespace fmm
