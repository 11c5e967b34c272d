// api.cu -- the extern "C" boundary declared in include/fmm.h.  Argument checking, plan lifetime, host-buffer
// convenience path; every computation is a kernel launched from plan.cu / evaluate.cu / m2l_fast.cu.
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <utility>

#include "internal.cuh"

namespace fmm {
namespace {
thread_local std::string g_err;
}
void set_error(const std::string& msg) { g_err = msg; }
}  // namespace fmm

struct fmm_plan {
    fmm::Plan P;
};

using namespace fmm;

namespace {

template <typename F>
fmm_status guarded(F&& f) {
    try {
        return f();
    } catch (CudaFail& c) {
        cudaGetLastError();  // clear the sticky-less error state
        return c.st;
    } catch (std::bad_alloc&) {
        set_error("host allocation failed");
        return FMM_ERR_ALLOC;
    } catch (...) {
        set_error("unexpected exception");
        return FMM_ERR_CUDA;
    }
}

size_t esize(fmm_dtype d) { return d == FMM_F32 ? 4 : 8; }

// per-device setup on plan creation: operator tables (device_ctx) and the memory pool -- keep up to 8 GiB of freed blocks mapped
// in the device's default memory pool (see DevBuf).  Returns the current device.
int init_device() {
    const int dev = current_device();
    DeviceCtx& ctx = device_ctx(dev);
    std::lock_guard<std::mutex> lock(ctx.mu);
    if (!ctx.pool_ready) {
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            unsigned long long thr = 8ull << 30;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        }
        cudaGetLastError();
        ctx.pool_ready = true;
    }
    return dev;
}

// every entry point that touches device memory of a plan: the plan's device must be the current one
bool on_plan_device(const Plan& P) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != P.device) {
        cudaGetLastError();
        set_error("the plan lives on device " + std::to_string(P.device) + " but the current device is " + std::to_string(dev) +
                  " (call cudaSetDevice first)");
        return false;
    }
    return true;
}

// N, p, N_max, s, dtype -> depth and box numbering of one hierarchy (rule T1 / T2); false if the tree is too large
bool init_shape(Plan& P, int64_t N, int p, int N_max, int s, fmm_dtype dtype, double theta) {
    P.N = N; P.p = p; P.N_max = N_max; P.s = s; P.dtype = dtype; P.theta = theta;
    P.K = (p + 1) * (p + 1);
    P.Kp = (P.K + 3) & ~3;
    int L = 0;  // smallest L with ceil(N / 2^(sL)) <= N_max
    for (;; ++L) {
        int64_t q = N;
        for (int i = 0; i < s * L; ++i) q = (q + 1) / 2;
        if (q <= N_max) break;
    }
    if ((int64_t)s * L > 30) { set_error("tree too deep: s*L > 30"); return false; }
    P.L = L;
    P.level_off.assign(L + 2, 0);
    for (int l = 0; l <= L; ++l) P.level_off[l + 1] = P.level_off[l] + ((int64_t)1 << (s * l));
    P.n_boxes = P.level_off[L + 1];
    P.n_leaves = (int64_t)1 << (s * L);
    if (P.n_boxes > 0x7fffff00ll) { set_error("too many boxes"); return false; }
    return true;
}

fmm_status copy_tree_impl(const Plan& P, int32_t* h_perm, int32_t* h_box_start, int32_t* h_box_count, void* h_box_lo, void* h_box_hi,
                          double* h_box_ctr, double* h_box_rad) {
    const size_t es = esize(P.dtype);
    FMM_CUDA_CHECK(cudaDeviceSynchronize());
    if (h_perm) FMM_CUDA_CHECK(cudaMemcpy(h_perm, P.perm.p, P.N * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (h_box_start) FMM_CUDA_CHECK(cudaMemcpy(h_box_start, P.box_start.p, P.n_boxes * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (h_box_count) FMM_CUDA_CHECK(cudaMemcpy(h_box_count, P.box_count.p, P.n_boxes * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (h_box_lo) FMM_CUDA_CHECK(cudaMemcpy(h_box_lo, P.box_lo.p, P.n_boxes * 3 * es, cudaMemcpyDeviceToHost));
    if (h_box_hi) FMM_CUDA_CHECK(cudaMemcpy(h_box_hi, P.box_hi.p, P.n_boxes * 3 * es, cudaMemcpyDeviceToHost));
    if (h_box_ctr) FMM_CUDA_CHECK(cudaMemcpy(h_box_ctr, P.box_ctr.p, P.n_boxes * 3 * sizeof(double), cudaMemcpyDeviceToHost));
    if (h_box_rad) FMM_CUDA_CHECK(cudaMemcpy(h_box_rad, P.box_rad.p, P.n_boxes * sizeof(double), cudaMemcpyDeviceToHost));
    return FMM_OK;
}

}  // namespace

extern "C" {

const char* fmm_last_error(void) { return g_err.c_str(); }
const char* fmm_version(void) { return "paper_2511_15269_b200 0.1 (sm_100a)"; }

fmm_status fmm_plan_create(const void* d_positions, int64_t N, int p, int N_max, int s, const fmm_admissibility* adm, fmm_dtype dtype,
                           void* cuda_stream, fmm_plan** out_plan) {
    if (out_plan) *out_plan = nullptr;
    return guarded([&]() -> fmm_status {
        g_err.clear();
        if (!out_plan || !d_positions) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (N < 1 || N > 0x7fffff00ll) { set_error("N must be in [1, 2^31)"); return FMM_ERR_INVALID_ARG; }
        if (p < 0 || p > PMAX) { set_error("p must be in [0, FMM_P_MAX]"); return FMM_ERR_INVALID_ARG; }
        if (N_max < 1 || s < 1) { set_error("N_max and s must be >= 1"); return FMM_ERR_INVALID_ARG; }
        if (dtype != FMM_F32 && dtype != FMM_F64) { set_error("unknown dtype"); return FMM_ERR_INVALID_ARG; }
        double theta = 0.77;
        int cross_level = 0;
        if (adm) {
            theta = adm->theta;
            cross_level = adm->cross_level;
            if (!(theta > 0.0 && theta < 1.0)) { set_error("theta must be in (0,1)"); return FMM_ERR_INVALID_ARG; }
            if (cross_level != 0 && cross_level != 1) { set_error("cross_level must be 0 or 1"); return FMM_ERR_INVALID_ARG; }
        }
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
            cudaGetLastError();
            set_error("no CUDA device: this library has no CPU fallback");
            return FMM_ERR_CUDA;
        }
        cudaStream_t st = (cudaStream_t)cuda_stream;
        const int dev = init_device();
        AllocScope scope(st);
        fmm_plan* h = new fmm_plan();
        Plan& P = h->P;
        try {
            P.device = dev;
            P.cross_level = cross_level;
            if (!init_shape(P, N, p, N_max, s, dtype, theta)) { delete h; return FMM_ERR_UNSUPPORTED; }
            cudaEvent_t e0, e1;
            FMM_CUDA_CHECK(cudaEventCreate(&e0));
            FMM_CUDA_CHECK(cudaEventCreate(&e1));
            FMM_CUDA_CHECK(cudaEventRecord(e0, st));
            build_tree(P, d_positions, st);
            build_lists(P, st);
            if (m2l_geo_wanted(p, dtype) && P.n_weak > 0) m2l_geo_prepare(P, st);
            const size_t es = esize(dtype);
            P.pq.alloc((size_t)N * 4 * es);
            P.near.alloc((size_t)N * 4 * es);
            P.Mc.alloc((size_t)P.n_boxes * P.Kp * es);
            P.Lc.alloc((size_t)P.n_boxes * P.Kp * es);
            FMM_CUDA_CHECK(cudaMemsetAsync(P.Mc.p, 0, P.Mc.n, st));
            FMM_CUDA_CHECK(cudaEventRecord(e1, st));
            FMM_CUDA_CHECK(cudaStreamSynchronize(st));
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            P.plan_ms[3] = ms;
            cudaEventDestroy(e0);
            cudaEventDestroy(e1);
        } catch (...) {
            delete h;
            throw;
        }
        *out_plan = h;
        return FMM_OK;
    });
}

fmm_status fmm_plan_create_targets(const void* d_sources, int64_t Ns, const void* d_targets, int64_t Nt, int p, int N_max, int s,
                                   const fmm_admissibility* adm, fmm_dtype dtype, void* cuda_stream, fmm_plan** out_plan) {
    if (out_plan) *out_plan = nullptr;
    return guarded([&]() -> fmm_status {
        g_err.clear();
        if (!out_plan || !d_sources || !d_targets) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (Ns < 1 || Ns > 0x7fffff00ll || Nt < 1 || Nt > 0x7fffff00ll) { set_error("Ns and Nt must be in [1, 2^31)"); return FMM_ERR_INVALID_ARG; }
        if (p < 0 || p > PMAX) { set_error("p must be in [0, FMM_P_MAX]"); return FMM_ERR_INVALID_ARG; }
        if (N_max < 1 || s < 1) { set_error("N_max and s must be >= 1"); return FMM_ERR_INVALID_ARG; }
        if (dtype != FMM_F32 && dtype != FMM_F64) { set_error("unknown dtype"); return FMM_ERR_INVALID_ARG; }
        double theta = 0.77;
        if (adm) {
            theta = adm->theta;  // cross_level is ignored: two hierarchies are always marched level by level
            if (!(theta > 0.0 && theta < 1.0)) { set_error("theta must be in (0,1)"); return FMM_ERR_INVALID_ARG; }
        }
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
            cudaGetLastError();
            set_error("no CUDA device: this library has no CPU fallback");
            return FMM_ERR_CUDA;
        }
        cudaStream_t st = (cudaStream_t)cuda_stream;
        const int dev = init_device();
        AllocScope scope(st);
        fmm_plan* h = new fmm_plan();
        Plan& P = h->P;
        try {
            P.device = dev;
            P.cross_level = 1;
            P.S.reset(new Plan());
            Plan& S = *P.S;
            S.device = dev;
            S.cross_level = 1;
            if (!init_shape(P, Nt, p, N_max, s, dtype, theta) || !init_shape(S, Ns, p, N_max, s, dtype, theta)) { delete h; return FMM_ERR_UNSUPPORTED; }
            cudaEvent_t e0, e1;
            FMM_CUDA_CHECK(cudaEventCreate(&e0));
            FMM_CUDA_CHECK(cudaEventCreate(&e1));
            FMM_CUDA_CHECK(cudaEventRecord(e0, st));
            build_tree(S, d_sources, st);
            const double sort_s = S.plan_ms[0], tree_s = S.plan_ms[1];
            build_tree(P, d_targets, st);
            P.plan_ms[0] += sort_s; P.plan_ms[1] += tree_s;
            build_lists(P, st);
            if (m2l_geo_wanted(p, dtype) && P.n_weak > 0) m2l_geo_prepare(P, st);
            const size_t es = esize(dtype);
            S.pq.alloc((size_t)Ns * 4 * es);
            S.Mc.alloc((size_t)S.n_boxes * S.Kp * es);
            FMM_CUDA_CHECK(cudaMemsetAsync(S.Mc.p, 0, S.Mc.n, st));
            P.pq.alloc((size_t)Nt * 4 * es);
            P.near.alloc((size_t)Nt * 4 * es);
            P.Lc.alloc((size_t)P.n_boxes * P.Kp * es);
            FMM_CUDA_CHECK(cudaEventRecord(e1, st));
            FMM_CUDA_CHECK(cudaStreamSynchronize(st));
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            P.plan_ms[3] = ms;
            cudaEventDestroy(e0);
            cudaEventDestroy(e1);
        } catch (...) {
            delete h;
            throw;
        }
        *out_plan = h;
        return FMM_OK;
    });
}

fmm_status fmm_plan_update(fmm_plan* plan, const void* d_positions, const void* d_targets, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        g_err.clear();
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        Plan& P = plan->P;
        if (!on_plan_device(P)) return FMM_ERR_INVALID_ARG;
        if (!P.S && (!d_positions || d_targets)) { set_error("a plan over one point set takes d_positions and d_targets == NULL"); return FMM_ERR_INVALID_ARG; }
        if (P.S && !d_positions && !d_targets) { set_error("nothing to update"); return FMM_ERR_INVALID_ARG; }
        cudaStream_t st = (cudaStream_t)cuda_stream;
        AllocScope scope(st);
        FMM_CUDA_CHECK(cudaDeviceSynchronize());  // no evaluate of this plan may still be reading the arrays that are rebuilt
        cudaEvent_t e0, e1;
        FMM_CUDA_CHECK(cudaEventCreate(&e0));
        FMM_CUDA_CHECK(cudaEventCreate(&e1));
        FMM_CUDA_CHECK(cudaEventRecord(e0, st));
        P.adj.reset();  // the transposed lists belong to the old positions
        P.shard_cache = Plan::Shard();
        ++P.epoch;      // captured evaluate graphs point into arrays that are reallocated below
        double sort_ms = 0, tree_ms = 0;
        if (P.S) {
            if (d_positions) { build_tree(*P.S, d_positions, st); sort_ms += P.S->plan_ms[0]; tree_ms += P.S->plan_ms[1]; }
            if (d_targets) { build_tree(P, d_targets, st); sort_ms += P.plan_ms[0]; tree_ms += P.plan_ms[1]; }
        } else {
            build_tree(P, d_positions, st);
            sort_ms = P.plan_ms[0]; tree_ms = P.plan_ms[1];
        }
        P.plan_ms[0] = sort_ms; P.plan_ms[1] = tree_ms;
        build_lists(P, st);
        if (m2l_geo_wanted(P.p, P.dtype) && P.n_weak > 0) m2l_geo_prepare(P, st);
        else P.m2l_geo.release();
        FMM_CUDA_CHECK(cudaEventRecord(e1, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        P.plan_ms[3] = ms;
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
        return FMM_OK;
    });
}

fmm_status fmm_plan_source_info(const fmm_plan* plan, int64_t* Ns, int* L, int64_t* n_boxes, int64_t* n_leaves) {
    if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
    const Plan& S = plan->P.S ? *plan->P.S : plan->P;
    if (Ns) *Ns = S.N;
    if (L) *L = S.L;
    if (n_boxes) *n_boxes = S.n_boxes;
    if (n_leaves) *n_leaves = S.n_leaves;
    return FMM_OK;
}

fmm_status fmm_plan_copy_source_tree(const fmm_plan* plan, int32_t* h_perm, int32_t* h_box_start, int32_t* h_box_count, void* h_box_lo,
                                     void* h_box_hi, double* h_box_ctr, double* h_box_rad) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        return copy_tree_impl(plan->P.S ? *plan->P.S : plan->P, h_perm, h_box_start, h_box_count, h_box_lo, h_box_hi, h_box_ctr, h_box_rad);
    });
}

fmm_status fmm_plan_copy_march(const fmm_plan* plan, int32_t* h_steps, int32_t* n_steps) {
    if (!plan || !n_steps) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
    const std::vector<int>& m = plan->P.march_steps;
    *n_steps = (int32_t)(m.size() / 2);
    if (h_steps) for (size_t i = 0; i < m.size(); ++i) h_steps[i] = m[i];
    return FMM_OK;
}

fmm_status fmm_plan_destroy(fmm_plan* plan) {
    if (!plan) return FMM_OK;
    return guarded([&]() -> fmm_status {
        // the plan's memory goes back to the pool of ITS device: switch to it for the duration of the call if necessary
        int cur = -1;
        const int pdev = plan->P.device;
        const bool have = cudaGetDevice(&cur) == cudaSuccess;
        if (have && cur != pdev) cudaSetDevice(pdev);
        cudaDeviceSynchronize();  // nothing of the plan may still be in flight on any stream when its memory returns to the pool
        delete plan;
        if (have && cur != pdev) cudaSetDevice(cur);
        cudaGetLastError();
        return FMM_OK;
    });
}

fmm_status fmm_evaluate(const fmm_plan* plan, const void* d_charges, void* d_potential, void* d_field, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan || !d_charges) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        AllocScope scope((cudaStream_t)cuda_stream);
        run_evaluate(plan->P, d_charges, d_potential, d_field, (cudaStream_t)cuda_stream, nullptr);
        return FMM_OK;
    });
}

fmm_status fmm_evaluate_adjoint(fmm_plan* plan, const void* d_cotangent_potential, const void* d_cotangent_field, void* d_charge_grad, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan || !d_charge_grad || (!d_cotangent_potential && !d_cotangent_field)) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        Plan& P = plan->P;
        if (!on_plan_device(P)) return FMM_ERR_INVALID_ARG;
        cudaStream_t st = (cudaStream_t)cuda_stream;
        AllocScope scope(st);
        // one point set with same-level lists: the lists are symmetric and the FMM potential operator is its own transpose
        // (M2M^T = L2L, M2L(t<-s)^T = M2L(s<-t), P2M^T = L2P in the normalised basis), so the plan is its own adjoint view
        const bool self_adjoint = !P.S && !P.cross_level;
        if (!self_adjoint) build_adjoint_view(P, st);
        const Plan& V = self_adjoint ? P : *P.adj;
        if (!self_adjoint) { P.adj->m2l_variant = P.m2l_variant; P.adj->serial = P.serial; P.adj->use_graph = P.use_graph; }
        run_evaluate(V, d_cotangent_potential, d_charge_grad, nullptr, st, nullptr, d_cotangent_field);
        return FMM_OK;
    });
}

fmm_status fmm_shard_box_range(int L, int s, int n_shards, int shard, int level, int64_t* h_begin, int64_t* h_end) {
    if (L < 0 || s < 1 || (int64_t)s * L > 30 || n_shards < 1 || shard < 0 || shard >= n_shards || level < 0 || level > L || !h_begin || !h_end) {
        set_error("bad argument");
        return FMM_ERR_INVALID_ARG;
    }
    shard_box_range(L, s, n_shards, shard, level, h_begin, h_end);
    return FMM_OK;
}

fmm_status fmm_evaluate_shard_upward(const fmm_plan* plan, int n_shards, int shard, const void* d_charges, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan || !d_charges) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        AllocScope scope((cudaStream_t)cuda_stream);
        run_shard_upward(plan->P, n_shards, shard, d_charges, (cudaStream_t)cuda_stream);
        return FMM_OK;
    });
}

fmm_status fmm_evaluate_shard_downward(const fmm_plan* plan, int n_shards, int shard, void* d_potential, void* d_field, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        AllocScope scope((cudaStream_t)cuda_stream);
        run_shard_downward(plan->P, n_shards, shard, d_potential, d_field, (cudaStream_t)cuda_stream);
        return FMM_OK;
    });
}

fmm_status fmm_plan_leaf_multipoles(const fmm_plan* plan, int copy_in, int64_t leaf_begin, int64_t leaf_end, void* d_rows, int64_t* h_row_elems,
                                    void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        const Plan& P = plan->P;
        if (P.S) { set_error("plans with separate targets are not supported"); return FMM_ERR_UNSUPPORTED; }
        if (h_row_elems) *h_row_elems = P.Kp;
        if (!d_rows) return FMM_OK;  // query only
        if (!on_plan_device(P)) return FMM_ERR_INVALID_ARG;
        if (leaf_begin < 0 || leaf_end > P.n_leaves || leaf_begin > leaf_end) { set_error("leaf range out of bounds"); return FMM_ERR_INVALID_ARG; }
        const size_t es = esize(P.dtype), row = (size_t)P.Kp * es;
        char* blk = P.Mc.p + ((size_t)P.level_off[P.L] + (size_t)leaf_begin) * row;
        const size_t bytes = (size_t)(leaf_end - leaf_begin) * row;
        if (bytes) FMM_CUDA_CHECK(cudaMemcpyAsync(copy_in ? (void*)blk : d_rows, copy_in ? (const void*)d_rows : (const void*)blk, bytes, cudaMemcpyDeviceToDevice,
                                                  (cudaStream_t)cuda_stream));
        return FMM_OK;
    });
}

fmm_status fmm_leaf_multipoles_noalloc(const fmm_plan* plan, const void* d_charges, void* d_rows, int64_t* h_row_elems, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        const Plan& P = plan->P;
        if (P.S) { set_error("plans with separate targets are not supported"); return FMM_ERR_UNSUPPORTED; }
        if (h_row_elems) *h_row_elems = P.Kp;
        if (!d_charges && !d_rows) return FMM_OK;  // query only
        if (!d_charges || !d_rows) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(P)) return FMM_ERR_INVALID_ARG;
        run_leaf_multipoles_noalloc(P, d_charges, d_rows, (cudaStream_t)cuda_stream);  // no AllocScope: nothing is allocated
        return FMM_OK;
    });
}

fmm_status fmm_evaluate_profiled(const fmm_plan* plan, const void* d_charges, void* d_potential, void* d_field, void* cuda_stream,
                                 double* h_stage_ms) {
    return guarded([&]() -> fmm_status {
        if (!plan || !d_charges || !h_stage_ms) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        cudaEvent_t ev[8];
        for (auto& e : ev) FMM_CUDA_CHECK(cudaEventCreate(&e));
        cudaStream_t st = (cudaStream_t)cuda_stream;
        AllocScope scope(st);
        run_evaluate(plan->P, d_charges, d_potential, d_field, st, ev);
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        for (int i = 0; i < 7; ++i) {
            float ms = 0;
            cudaEventElapsedTime(&ms, ev[i], ev[i + 1]);
            h_stage_ms[i] = ms;
        }
        std::swap(h_stage_ms[5], h_stage_ms[6]);  // launched P2P, then L2P (+finalize); reported as [5] L2P, [6] P2P
        float tot = 0;
        cudaEventElapsedTime(&tot, ev[0], ev[7]);
        h_stage_ms[7] = tot;
        for (auto& e : ev) cudaEventDestroy(e);
        return FMM_OK;
    });
}

fmm_status fmm_evaluate_host(const fmm_plan* plan, const void* h_charges, void* h_potential, void* h_field, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan || !h_charges) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        Plan& P = const_cast<Plan&>(plan->P);
        const size_t es = esize(P.dtype);
        cudaStream_t st = (cudaStream_t)cuda_stream;
        AllocScope scope(st);
        const int64_t Nq = P.S ? P.S->N : P.N;  // charges live on the sources
        if (!P.h2d_q.p) P.h2d_q.alloc((size_t)Nq * es);
        if (!P.d2h_out.p) P.d2h_out.alloc((size_t)P.N * 4 * es);
        FMM_CUDA_CHECK(cudaMemcpyAsync(P.h2d_q.p, h_charges, (size_t)Nq * es, cudaMemcpyHostToDevice, st));
        char* dpot = h_potential ? P.d2h_out.p : nullptr;
        char* dfld = h_field ? P.d2h_out.p + (size_t)P.N * es : nullptr;
        run_evaluate(P, P.h2d_q.p, dpot, dfld, st, nullptr);
        if (h_potential) FMM_CUDA_CHECK(cudaMemcpyAsync(h_potential, dpot, (size_t)P.N * es, cudaMemcpyDeviceToHost, st));
        if (h_field) FMM_CUDA_CHECK(cudaMemcpyAsync(h_field, dfld, (size_t)P.N * 3 * es, cudaMemcpyDeviceToHost, st));
        FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        return FMM_OK;
    });
}

fmm_status fmm_evaluate_host_submit(const fmm_plan* plan, const void* h_charges, void* h_potential, void* h_field, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan || !h_charges) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        Plan& P = const_cast<Plan&>(plan->P);
        if (P.hs_count >= 2) { set_error("two submitted calls are in flight: call fmm_evaluate_host_wait first"); return FMM_ERR_UNSUPPORTED; }
        const size_t es = esize(P.dtype);
        cudaStream_t st = (cudaStream_t)cuda_stream;
        AllocScope scope(st);
        const int64_t Nq = P.S ? P.S->N : P.N;
        Plan::HostSlot& h = P.hslot[(P.hs_head + P.hs_count) & 1];
        if (!P.s_h2d) {
            FMM_CUDA_CHECK(cudaStreamCreateWithFlags(&P.s_h2d, cudaStreamNonBlocking));
            FMM_CUDA_CHECK(cudaStreamCreateWithFlags(&P.s_d2h, cudaStreamNonBlocking));
        }
        if (!h.q.p) {  // first use of the slot: its buffers come from the pool on st and are used on the copy streams
            h.q.alloc((size_t)Nq * es);
            h.out.alloc((size_t)P.N * 4 * es);
            for (cudaEvent_t* e : {&h.e_in, &h.e_eval, &h.e_out}) FMM_CUDA_CHECK(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
            FMM_CUDA_CHECK(cudaStreamSynchronize(st));
        }
        // charges in, beside whatever st is still computing (the slot's previous call has been waited for)
        FMM_CUDA_CHECK(cudaMemcpyAsync(h.q.p, h_charges, (size_t)Nq * es, cudaMemcpyHostToDevice, P.s_h2d));
        FMM_CUDA_CHECK(cudaEventRecord(h.e_in, P.s_h2d));
        FMM_CUDA_CHECK(cudaStreamWaitEvent(st, h.e_in, 0));
        char* dpot = h_potential ? h.out.p : nullptr;
        char* dfld = h_field ? h.out.p + (size_t)P.N * es : nullptr;
        run_evaluate(P, h.q.p, dpot, dfld, st, nullptr);
        FMM_CUDA_CHECK(cudaEventRecord(h.e_eval, st));
        // results out, beside the next call's evaluate
        FMM_CUDA_CHECK(cudaStreamWaitEvent(P.s_d2h, h.e_eval, 0));
        if (h_potential) FMM_CUDA_CHECK(cudaMemcpyAsync(h_potential, dpot, (size_t)P.N * es, cudaMemcpyDeviceToHost, P.s_d2h));
        if (h_field) FMM_CUDA_CHECK(cudaMemcpyAsync(h_field, dfld, (size_t)P.N * 3 * es, cudaMemcpyDeviceToHost, P.s_d2h));
        FMM_CUDA_CHECK(cudaEventRecord(h.e_out, P.s_d2h));
        ++P.hs_count;
        return FMM_OK;
    });
}

fmm_status fmm_evaluate_host_wait(const fmm_plan* plan) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        Plan& P = const_cast<Plan&>(plan->P);
        if (P.hs_count == 0) { set_error("no submitted call is in flight"); return FMM_ERR_INVALID_ARG; }
        FMM_CUDA_CHECK(cudaEventSynchronize(P.hslot[P.hs_head].e_out));
        P.hs_head ^= 1;
        --P.hs_count;
        return FMM_OK;
    });
}

fmm_status fmm_plan_info(const fmm_plan* plan, int* L, int64_t* n_boxes, int64_t* n_leaves, int64_t* n_weak, int64_t* n_strong,
                         int64_t* n_p2p_pairs) {
    if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
    const Plan& P = plan->P;
    if (L) *L = P.L;
    if (n_boxes) *n_boxes = P.n_boxes;
    if (n_leaves) *n_leaves = P.n_leaves;
    if (n_weak) *n_weak = P.n_weak;
    if (n_strong) *n_strong = P.n_strong;
    if (n_p2p_pairs) *n_p2p_pairs = P.n_p2p_pairs;
    return FMM_OK;
}

fmm_status fmm_plan_copy_tree(const fmm_plan* plan, int32_t* h_perm, int32_t* h_box_start, int32_t* h_box_count, void* h_box_lo,
                              void* h_box_hi, double* h_box_ctr, double* h_box_rad) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        if (!on_plan_device(plan->P)) return FMM_ERR_INVALID_ARG;
        return copy_tree_impl(plan->P, h_perm, h_box_start, h_box_count, h_box_lo, h_box_hi, h_box_ctr, h_box_rad);
    });
}

fmm_status fmm_plan_copy_lists(const fmm_plan* plan, int64_t* h_weak_off, int32_t* h_weak_src, int64_t* h_strong_off, int32_t* h_strong_src) {
    return guarded([&]() -> fmm_status {
        if (!plan) { set_error("NULL plan"); return FMM_ERR_INVALID_ARG; }
        const Plan& P = plan->P;
        if (!on_plan_device(P)) return FMM_ERR_INVALID_ARG;
        FMM_CUDA_CHECK(cudaDeviceSynchronize());
        if (h_weak_off) FMM_CUDA_CHECK(cudaMemcpy(h_weak_off, P.weak_off.p, (P.n_boxes + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost));
        if (h_weak_src && P.n_weak) FMM_CUDA_CHECK(cudaMemcpy(h_weak_src, P.weak_src.p, P.n_weak * sizeof(int32_t), cudaMemcpyDeviceToHost));
        if (h_strong_off) FMM_CUDA_CHECK(cudaMemcpy(h_strong_off, P.strong_off.p, (P.n_leaves + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost));
        if (h_strong_src && P.n_strong) FMM_CUDA_CHECK(cudaMemcpy(h_strong_src, P.strong_src.p, P.n_strong * sizeof(int32_t), cudaMemcpyDeviceToHost));
        return FMM_OK;
    });
}

fmm_status fmm_plan_timings(const fmm_plan* plan, double* h_ms) {
    if (!plan || !h_ms) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
    for (int i = 0; i < 4; ++i) h_ms[i] = plan->P.plan_ms[i];
    return FMM_OK;
}

fmm_status fmm_plan_launches(const fmm_plan* plan, int64_t* h) {
    if (!plan || !h) { set_error("NULL pointer argument"); return FMM_ERR_INVALID_ARG; }
    *h = evaluate_launches(plan->P);
    return FMM_OK;
}

fmm_status fmm_translation_work(int p, fmm_dtype dtype, int kind, int64_t* h_fma, int64_t* h_mul, int64_t* h_add) {
    if (p < 0 || p > PMAX || kind < 0 || kind > 2 || (dtype != FMM_F32 && dtype != FMM_F64)) { set_error("bad argument"); return FMM_ERR_INVALID_ARG; }
    int64_t w[3];
    xlate_work(p, dtype, kind, w);
    if (h_fma) *h_fma = w[0];
    if (h_mul) *h_mul = w[1];
    if (h_add) *h_add = w[2];
    return FMM_OK;
}

fmm_status fmm_plan_set_schedule(fmm_plan* plan, int serial) {
    if (!plan || serial < 0 || serial > 1) { set_error("bad argument"); return FMM_ERR_INVALID_ARG; }
    plan->P.serial = serial != 0;
    return FMM_OK;
}

fmm_status fmm_plan_set_deterministic(fmm_plan* plan, int on, void* cuda_stream) {
    return guarded([&]() -> fmm_status {
        if (!plan || on < 0 || on > 1) { set_error("bad argument"); return FMM_ERR_INVALID_ARG; }
        Plan& P = plan->P;
        if (!on_plan_device(P)) return FMM_ERR_INVALID_ARG;
        if (P.s > 5) { set_error("deterministic mode needs s <= 5 (the children of a box must fit one warp)"); return FMM_ERR_UNSUPPORTED; }
        if (P.deterministic == (on != 0)) return FMM_OK;
        cudaStream_t st = (cudaStream_t)cuda_stream;
        AllocScope scope(st);
        FMM_CUDA_CHECK(cudaDeviceSynchronize());
        P.deterministic = on != 0;
        ++P.epoch;
        // one P2P work item per leaf (no partial sums combined with atomics) / the load-balanced segments again
        if (P.n_leaves > 0 && P.strong_off.p) build_p2p_items(P, st, P.deterministic);
        P.shard_cache = Plan::Shard();
        P.adj.reset();
        return FMM_OK;
    });
}

fmm_status fmm_plan_set_graph(fmm_plan* plan, int on) {
    if (!plan || on < 0 || on > 2) { set_error("bad argument"); return FMM_ERR_INVALID_ARG; }
    plan->P.use_graph = on;
    if (plan->P.adj) plan->P.adj->use_graph = on;
    return FMM_OK;
}

fmm_status fmm_plan_set_m2l_variant(fmm_plan* plan, int variant) {
    if (!plan || variant < 0 || variant > 1) { set_error("bad argument"); return FMM_ERR_INVALID_ARG; }
    plan->P.m2l_variant = variant;
    return FMM_OK;
}

}  // extern "C"
