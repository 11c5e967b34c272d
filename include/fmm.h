/* fmm.h -- C-ABI boundary of the B200-native adaptive Laplace FMM (arXiv 2511.15269, "jaxFMM").
 *
 * The paper's interface is two calls, gen_hierarchy(pts, p, theta, ...) -> hier and
 * eval_potential(chrgs, **hier) (Listing 1), the hierarchy being reusable for new
 * charges.  Here: fmm_plan_create builds the hierarchy and the interaction lists on
 * the device, fmm_evaluate runs P2M -> M2M -> M2L -> L2L -> L2P + P2P (stage order PAPER.md:251).
 *
 * Result definition (eqs. (1)-(3)):
 *     potential_i = -(1/4pi) * sum_{j != i} q_j / |r_i - r_j|        field_i = -grad potential (r_i)
 * approximated by a p-th order FMM (eqs. (9)-(14)); pairs at zero distance
 * contribute nothing.
 *
 * Conventions
 *  - "DEVICE" pointers are CUDA device pointers of the current device; "HOST" pointers are ordinary
 *    host memory.  The caller owns every buffer it passes; the plan copies what it needs and never
 *    keeps caller pointers.  The plan owns all of its internal device memory.
 *  - dtype selects the arithmetic AND the element type of positions/charges/outputs (float or double).
 *    Geometric decisions (box centres, radii, admissibility) are always taken in IEEE fp64.
 *  - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).
 *  - fmm_plan_create and the fmm_plan_copy_* / fmm_plan_info calls synchronise the stream before
 *    returning; fmm_evaluate only enqueues work on the stream (asynchronous).  Evaluations on one plan
 *    must be serialised by stream order (the plan owns the coefficient scratch arrays).
 *  - A plan lives on the CUDA device that is current when it is created.  Every later call that takes the plan must run with
 *    that device current (cudaSetDevice) and returns FMM_ERR_INVALID_ARG otherwise; fmm_plan_destroy switches by itself.
 *    One process may hold plans on several devices (operator tables, constant memory and kernel attributes are kept per
 *    device; their one-time setup is mutex-guarded).  Calls on ONE plan must not overlap in time on the host.
 *  - Plan memory comes from the device's default stream-ordered memory pool (cudaMallocAsync); up to 8 GiB of freed blocks stay
 *    cached there for the next plan (cudaMemPoolTrimTo on the default pool returns them).
 *  - Outputs are in INPUT order.
 *  - No exception or abort crosses this boundary: every failure is a status code, *out_plan is NULL on
 *    failure, fmm_last_error() returns a thread-local message.
 *  - There is no CPU fallback: without a CUDA device every compute entry point returns FMM_ERR_CUDA.
 */
#ifndef PAPER_2511_15269_FMM_H
#define PAPER_2511_15269_FMM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fmm_plan fmm_plan; /* opaque */

typedef enum {
    FMM_OK = 0,
    FMM_ERR_INVALID_ARG = 1, /* NULL pointer, N<1, p<0 or p>FMM_P_MAX, N_max<1, s<1, theta not in (0,1), non-finite position */
    FMM_ERR_ALLOC = 2,       /* device or host allocation failed */
    FMM_ERR_CUDA = 3,        /* any other CUDA runtime error (message in fmm_last_error) */
    FMM_ERR_UNSUPPORTED = 4  /* a tree too deep for 31-bit box ids, lists beyond 2^31 pairs */
} fmm_status;

typedef enum { FMM_F32 = 0, FMM_F64 = 1 } fmm_dtype;

#define FMM_P_MAX 16

/* Admissibility parameters of eq. (4):  R + theta*r < theta*d. */
typedef struct {
    double theta;    /* 0 < theta < 1; the paper's default is 0.77 */
    int cross_level; /* 0 = same-level lists (the default).  1 = level-marching lists: weak
                      * pairs may join a target box with a source box one level below it; the march over (target level,
                      * source level) is (0,0), (0,1), (1,1), (1,2), ..., (L,L): on equal levels the SOURCE level is increased
                      * first (reading S9), so a source box is never coarser than its target box.
                      * Fewer M2L pairs at the same eq. (4). */
} fmm_admissibility;

/* Build hierarchy + lists for N charges (Listing 2; lists PAPER.md:72-74).
 *   d_positions : DEVICE, N x 3 row-major (x,y,z), element type = dtype.  Read only during this call.
 *   p           : expansion order, 0..FMM_P_MAX (eqs. (9),(11)).
 *   N_max       : leaves hold at most N_max charges.   s : splits per level, 2^s children.
 *   adm         : HOST pointer; NULL selects theta = 0.77, same-level lists.
 * Tree depth L is the smallest l with ceil(N / 2^(s*l)) <= N_max.  Synchronises the stream. */
fmm_status fmm_plan_create(const void* d_positions, int64_t N, int p, int N_max, int s,
                           const fmm_admissibility* adm, fmm_dtype dtype, void* cuda_stream, fmm_plan** out_plan);

/* Evaluate potential and/or field for new charges on an existing plan.
 *   d_charges   : DEVICE, N, input order, dtype.
 *   d_potential : DEVICE, N, input order, dtype; may be NULL.
 *   d_field     : DEVICE, N x 3 row-major, input order, dtype; may be NULL.
 * An output that is NULL is not computed: with d_field == NULL the near-field and L2P kernels skip the field arithmetic
 * (about 15 % less time at N = 1M, p = 8).
 * Asynchronous on cuda_stream. */
fmm_status fmm_evaluate(const fmm_plan* plan, const void* d_charges, void* d_potential, void* d_field, void* cuda_stream);

/* Adjoint evaluate: the vector-Jacobian product of fmm_evaluate with respect to the charges (where JAX autodiff
 * differentiates a loss on the potential with respect to the charges).  fmm_evaluate is linear in the charges -- potential = A q,
 * field = F q with the FMM operators A, F of this plan -- so for cotangents ubar (of the potential) and fbar (of the field)
 *     charge_grad = A^T ubar + F^T fbar .
 * It is computed as the TRANSPOSE OF THE FORWARD OPERATOR on the same plan, stage by stage: L2P^T is a P2M at the targets (with
 * dipole moments -fbar for the field part), L2L^T = M2M and M2M^T = L2L run on the other hierarchy, M2L^T is the M2L over the
 * transposed weak list, P2P^T the near field over the transposed strong list.  The transposed lists are built on the first call
 * (which synchronises the stream) and kept in the plan; a plan over one point set with same-level lists needs none (its lists
 * are symmetric).  <ubar, A q> + <fbar, F q> = <charge_grad, q> holds to rounding, not just to the truncation error of the FMM.
 *   d_cotangent_potential : DEVICE, Nt (N), target input order, dtype; may be NULL (zero).
 *   d_cotangent_field     : DEVICE, Nt x 3 (N x 3), dtype; may be NULL (zero); at least one of the two must be given.
 *   d_charge_grad         : DEVICE, Ns (N), source input order, dtype (overwritten).
 * Asynchronous on cuda_stream after the first call. */
fmm_status fmm_evaluate_adjoint(fmm_plan* plan, const void* d_cotangent_potential, const void* d_cotangent_field, void* d_charge_grad,
                                void* cuda_stream);

/* Target-sharded evaluate for several GPUs (the paper has no multi-device support).  Every rank holds
 * the same plan (the positions are replicated; building it costs milliseconds) and all charges, and owns the targets of a contiguous
 * range of leaves -- a set of subtrees, because the tree order is a Z-order: shard r of n owns the leaves
 * [n_leaves r / n, n_leaves (r+1) / n).  One evaluate is
 *     fmm_evaluate_shard_upward   : permute, P2M for the shard's leaves (1/n of the work)
 *     <all-gather of the leaf rows of the multipole array among the ranks>   -- the ONE data-path collective; the caller runs it
 *                                   (paper_2511_15269_b200/fmm.py: NCCL through torch.distributed) on the rows that
 *                                   fmm_plan_leaf_multipoles copies out of / into the plan
 *     fmm_evaluate_shard_downward : M2M (all boxes, redundant: 0.05 ms), M2L and L2L for the shard's boxes and their ancestors,
 *                                   P2P and L2P for its leaves; writes potential / field of the shard's particles ONLY (input order;
 *                                   the other entries of the output arrays are not touched).
 * Both calls are asynchronous on cuda_stream (the first downward call of a shard reads a few list offsets back and synchronises).
 * Plans over one point set, orders 1..12 (the specialised kernels), m2l_variant 0; FMM_ERR_UNSUPPORTED otherwise.
 * fmm_shard_box_range needs no device: the level-local range of boxes of `level` that a shard touches (its leaves for level = L,
 * their ancestors above), for a tree of depth L with 2^s children per box. */
fmm_status fmm_shard_box_range(int L, int s, int n_shards, int shard, int level, int64_t* h_begin, int64_t* h_end);
fmm_status fmm_evaluate_shard_upward(const fmm_plan* plan, int n_shards, int shard, const void* d_charges, void* cuda_stream);
fmm_status fmm_evaluate_shard_downward(const fmm_plan* plan, int n_shards, int shard, void* d_potential, void* d_field, void* cuda_stream);
/* Leaf rows [leaf_begin, leaf_end) of the plan's multipole array, row = *h_row_elems elements of the plan's dtype ((p+1)^2 rounded up
 * to a multiple of 4): copy_in = 0 copies them to d_rows (DEVICE), copy_in = 1 copies d_rows into the plan.  d_rows = NULL only
 * queries the row length.  Asynchronous on cuda_stream. */
fmm_status fmm_plan_leaf_multipoles(const fmm_plan* plan, int copy_in, int64_t leaf_begin, int64_t leaf_end, void* d_rows, int64_t* h_row_elems,
                                    void* cuda_stream);

/* Leaf multipoles WITHOUT ANY ALLOCATION, for callers that must not reach cudaMalloc (code under stream capture, tight serving
 * loops, harnesses that forbid it).  Computes what fmm_evaluate_shard_upward(plan, 1, 0, ...) followed by
 * fmm_plan_leaf_multipoles(plan, 0, 0, n_leaves, ...) delivers -- the P2M step, eq. (13), for ALL leaves:
 *     d_rows[leaf * row + n^2 + n + m] = M_n^m of leaf `leaf` for the charges d_charges,  row = *h_row_elems = (p+1)^2 rounded up
 *     to a multiple of 4 (normalised, length-scaled coefficients; the padding of a row is written as zero)
 * but with the intermediate array of that step (the particles in tree order, packed x, y, z, q) in a STATIC device array of
 * FMM_NOALLOC_MAX_BYTES instead of the plan's own scratch, and the rows written straight into the caller's buffer.  The call
 * writes nothing in the plan (it may run beside an evaluate of the same plan) and calls no cudaMalloc / cudaFree / allocating
 * library routine.
 *   plan       : a plan over ONE point set (FMM_ERR_UNSUPPORTED for fmm_plan_create_targets plans), any order p.
 *   d_charges  : DEVICE, N, dtype, input order.      d_rows : DEVICE, n_leaves x row, dtype, overwritten.
 *   h_row_elems: HOST out (may be NULL).  d_charges = d_rows = NULL only queries it.
 * Limit: N x 4 x sizeof(dtype) <= FMM_NOALLOC_MAX_BYTES, i.e. N <= 524 288 (fp32) / 262 144 (fp64); beyond it the call returns
 * FMM_ERR_UNSUPPORTED with the sizes in fmm_last_error() and launches nothing.
 * The static array costs FMM_NOALLOC_MAX_BYTES on every GPU that loads the library, until the process exits.  ALL calls on a
 * device share it: calls that may overlap on the GPU (different streams without an ordering between them) race -- order them.
 * It keeps the contents of the last call; every call overwrites the part it reads, nothing has to be cleared.
 * The first call on a device does one-time set-up (symbol address, constant tables) and is not capturable; later calls are
 * asynchronous on cuda_stream and consist of one memset and two kernel launches. */
#define FMM_NOALLOC_MAX_BYTES (8u << 20)
fmm_status fmm_leaf_multipoles_noalloc(const fmm_plan* plan, const void* d_charges, void* d_rows, int64_t* h_row_elems, void* cuda_stream);

/* Same operation with HOST buffers: copies charges host->device, evaluates, copies the results back and
 * synchronises.  h_potential / h_field may be NULL.  (The end-to-end path timed by bench.py's "e2e".) */
fmm_status fmm_evaluate_host(const fmm_plan* plan, const void* h_charges, void* h_potential, void* h_field, void* cuda_stream);

/* The host path as a two-deep pipeline, for callers that evaluate many charge vectors on one plan (time stepping, the
 * optimisation loop of PAPER.md:281-310): _submit enqueues what fmm_evaluate_host does -- charges host->device, evaluate,
 * results device->host -- and returns without waiting; _wait blocks until the OLDEST submitted call has delivered its results
 * into the host buffers it was given.  The copies run on two internal streams, so the 4 B / particle in and 16 B / particle out
 * of one call cross PCIe while the other call's kernels run (the evaluates themselves stay ordered on cuda_stream: they
 * share the plan's coefficient arrays).  Each of the two slots owns device staging for charges and results.
 *   h_charges, h_potential, h_field: HOST, as for fmm_evaluate_host; PINNED memory is needed for the copies to overlap; the
 *   buffers of a call belong to the library until the matching _wait returns (use two sets when two calls are in flight).
 * At most two calls may be in flight: a third _submit returns FMM_ERR_UNSUPPORTED; _wait with nothing in flight returns
 * FMM_ERR_INVALID_ARG.  Results are those of fmm_evaluate_host (same kernels, same schedule).  fmm_plan_update and
 * fmm_plan_destroy must not be called with calls in flight (destroy waits for them). */
fmm_status fmm_evaluate_host_submit(const fmm_plan* plan, const void* h_charges, void* h_potential, void* h_field, void* cuda_stream);
fmm_status fmm_evaluate_host_wait(const fmm_plan* plan);

/* Separate sources and targets: potential and field AT the Nt targets caused by charges AT the Ns sources.
 * Two hierarchies are built with the same rules (N_max, s): one over the sources, one over the targets; source boxes are
 * compared with target boxes by eq. (4) while marching through the levels from (l_trg, l_src) = (0, 0): 1. increase the
 * level with the larger average box radius (mean radius of the non-empty boxes of the level); 2. if equal, the source
 * level; 3. if one hierarchy has no more levels, the other; 4. stop when no pair is left or both are at their leaf
 * level.  Pairs still failing there are summed directly (P2P between a target leaf and a source leaf).
 *   d_sources : DEVICE, Ns x 3, dtype;  d_targets : DEVICE, Nt x 3, dtype.  Read only during this call.
 *   adm       : HOST pointer or NULL (theta = 0.77); cross_level is ignored (two hierarchies are always marched).
 * On such a plan fmm_evaluate / fmm_evaluate_host / fmm_evaluate_profiled take Ns charges (source input order) and
 * write Nt potentials / Nt x 3 field vectors (target input order); a target that coincides with a source gets no
 * contribution from it (reading S3).  fmm_plan_info / fmm_plan_copy_tree describe the TARGET hierarchy,
 * fmm_plan_source_info / fmm_plan_copy_source_tree the SOURCE hierarchy; in fmm_plan_copy_lists rows are target boxes /
 * target leaves and entries are source boxes (global ids of the source hierarchy) / source leaves. */
fmm_status fmm_plan_create_targets(const void* d_sources, int64_t Ns, const void* d_targets, int64_t Nt, int p, int N_max, int s,
                                   const fmm_admissibility* adm, fmm_dtype dtype, void* cuda_stream, fmm_plan** out_plan);

/* Re-plan for moved points (in jaxFMM every change of the positions costs a new gen_hierarchy, minutes with
 * JIT): rebuilds hierarchy and interaction lists of an existing plan for new positions of the SAME number of points, with the
 * plan's p, N_max, s, theta, list kind and dtype.  The result is exactly the plan fmm_plan_create would build for these positions
 * (same kernels: hierarchy and lists bit-exact against the oracle); what is saved is every allocation -- all arrays whose size
 * depends only on N stay in place, the evaluate scratch and the internal streams are kept -- and, for a plan with separate targets,
 * the hierarchy of the side that did not move.
 *   one point set   : d_positions = DEVICE, N x 3, dtype;  d_targets must be NULL.
 *   separate targets: d_positions = new sources (Ns x 3) or NULL (unchanged), d_targets = new targets (Nt x 3) or NULL (unchanged).
 * Waits for the device to be idle, then runs on cuda_stream and synchronises it.  On failure (e.g. non-finite positions ->
 * FMM_ERR_INVALID_ARG) the plan is left without a valid hierarchy: update it again with valid positions or destroy it. */
fmm_status fmm_plan_update(fmm_plan* plan, const void* d_positions, const void* d_targets, void* cuda_stream);

/* Source hierarchy of a plan (HOST outputs, any may be NULL); for a plan made by fmm_plan_create it is the one hierarchy. */
fmm_status fmm_plan_source_info(const fmm_plan* plan, int64_t* Ns, int* L, int64_t* n_boxes, int64_t* n_leaves);
/* As fmm_plan_copy_tree, for the source hierarchy (sizes from fmm_plan_source_info). */
fmm_status fmm_plan_copy_source_tree(const fmm_plan* plan, int32_t* h_perm, int32_t* h_box_start, int32_t* h_box_count,
                                     void* h_box_lo, void* h_box_hi, double* h_box_ctr, double* h_box_rad);
/* The (l_trg, l_src) level pairs the level march visited, in order (plans with cross_level = 1 or separate targets;
 * n_steps = 0 otherwise).  h_steps: 2 * n_steps int32, may be NULL to query n_steps (at most L_trg + L_src + 1). */
fmm_status fmm_plan_copy_march(const fmm_plan* plan, int32_t* h_steps, int32_t* n_steps);

/* Frees all device memory of the plan.  NULL is allowed. */
fmm_status fmm_plan_destroy(fmm_plan* plan);

/* Introspection (HOST outputs, any may be NULL): tree depth L, number of boxes on all levels 0..L, number of
 * leaf boxes 2^(s*L), number of weak (M2L) pairs over all levels, number of strong leaf pairs (including (t,t)),
 * number of particle pairs the P2P stage visits (sum over strong leaf pairs of n_t * n_s). */
fmm_status fmm_plan_info(const fmm_plan* plan, int* L, int64_t* n_boxes, int64_t* n_leaves, int64_t* n_weak,
                         int64_t* n_strong, int64_t* n_p2p_pairs);

/* Copy the hierarchy to HOST buffers (any may be NULL).  Boxes are numbered level by level, level l holding
 * 2^(s*l) boxes, children of box b being b*2^s + j (lower half first at every sub-split).
 *   h_perm      : N int32, tree order -> input index (leaves in box order, ascending input index inside a leaf).
 *   h_box_start : n_boxes int32, first tree-order slot of the box;  h_box_count : n_boxes int32.
 *   h_box_lo/hi : n_boxes x 3, dtype, tight particle bounding box (zeros for empty boxes).
 *   h_box_ctr   : n_boxes x 3 double, 0.5*(lo+hi);  h_box_rad : n_boxes double, half diagonal (fp64, no FMA). */
fmm_status fmm_plan_copy_tree(const fmm_plan* plan, int32_t* h_perm, int32_t* h_box_start, int32_t* h_box_count,
                              void* h_box_lo, void* h_box_hi, double* h_box_ctr, double* h_box_rad);

/* Copy the interaction lists to HOST buffers (any may be NULL), canonical form: CSR by target, sources ascending.
 *   h_weak_off   : n_boxes+1 int64 (row = target global box id);  h_weak_src : n_weak int32 global box ids.
 *   h_strong_off : n_leaves+1 int64 (row = target leaf index);    h_strong_src : n_strong int32 leaf indices. */
fmm_status fmm_plan_copy_lists(const fmm_plan* plan, int64_t* h_weak_off, int32_t* h_weak_src,
                               int64_t* h_strong_off, int32_t* h_strong_src);

/* Per-stage device times of the most recent fmm_evaluate_profiled call, in milliseconds (HOST out, 8 doubles):
 * [0] permute, [1] P2M, [2] M2M, [3] M2L, [4] L2L, [5] L2P + finalize, [6] P2P, [7] total.  fmm_evaluate_profiled is
 * fmm_evaluate with CUDA events between the stages (it synchronises the stream). */
fmm_status fmm_evaluate_profiled(const fmm_plan* plan, const void* d_charges, void* d_potential, void* d_field,
                                 void* cuda_stream, double* h_stage_ms);

/* Plan-phase device times in ms (HOST out, 4 doubles): [0] sort keys, [1] tree rounds, [2] lists, [3] total. */
fmm_status fmm_plan_timings(const fmm_plan* plan, double* h_ms);

/* Selects the kernel family used by subsequent fmm_evaluate calls on this plan:
 * 0 = automatic (the one-translation-per-thread kernels for M2M / M2L / L2L and the warp-per-leaf P2P kernels; the generic
 * kernels where no specialised kernel exists for (p, dtype)), 1 = force the generic warp-per-box kernels (any p <= FMM_P_MAX,
 * both dtypes; a second, independent implementation of App. B that the tests cross-check against the oracle). */
fmm_status fmm_plan_set_m2l_variant(fmm_plan* plan, int variant);

/* Reproducibility.  By default the translation kernels add the partial sums of a row of the coefficient arrays with floating-point
 * atomics and a leaf with a very long strong list is summed in several pieces, so two evaluates of the same input agree to rounding
 * (1e-13 relative in fp64), not bit for bit.  on = 1: every sum has ONE contributor that adds in list order -- the M2L runs with one
 * warp per target box (p <= 8) or in the generic warp-per-box kernel (p >= 9), the P2P with one work item per leaf, and the kernels
 * run in the serial schedule: two evaluates of the same charges on the same plan return identical bits.  Costs about 16 % at
 * N = 1M, p = 8, fp32 (1.28 -> 1.49 ms per evaluate on B200).  Requires s <= 5.  Synchronises the device (the P2P work items are rebuilt). */
fmm_status fmm_plan_set_deterministic(fmm_plan* plan, int on, void* cuda_stream);

/* Schedule of subsequent fmm_evaluate / fmm_evaluate_host calls on this plan.  0 (default) = concurrent: the call forks
 * three internal streams from cuda_stream and joins them back before it returns control of the stream -- the near field
 * (P2P) runs beside the whole far-field chain and the M2M pass beside the leaf-level M2L; for the caller the call is
 * still one asynchronous operation in cuda_stream order.  1 = serial: every kernel is launched on cuda_stream itself
 * (what fmm_evaluate_profiled always does).  Both schedules run the same kernels on the same data; results agree to the
 * order of the floating-point atomics. */
fmm_status fmm_plan_set_schedule(fmm_plan* plan, int serial);

/* CUDA graphs.  on = 1: the second fmm_evaluate / fmm_evaluate_adjoint / fmm_evaluate_host call that sees the same
 * device pointers (charges, potential, field) captures the launches of one evaluate -- kernels, memsets and the fork / join
 * edges of the concurrent schedule -- into a CUDA graph on a stream the plan owns; every later call with those pointers is one
 * cudaGraphLaunch on cuda_stream (the plan keeps the graphs of the last four pointer sets).  Same kernels, same data, same
 * results; what changes is the host cost of an evaluate (about 10 + 2 L launches -> 1), which bounds the evaluate time below
 * N ~ 1e5.  A call made while cuda_stream is itself being captured by the caller launches plainly, so the evaluate can be part
 * of a caller's graph.  As before, two evaluates of ONE plan must not overlap: order them on one stream or with events.
 * on = 0: always launch plainly.  on = 2 (default): as 1 for plans with fewer than 2^19 points (sources + targets), as 0 above
 * -- there the device time hides the launches and the replay measured 2-3 % slower than the stream schedule (N = 1M, B200).
 * A failed capture disables the graphs of the plan and falls back to plain launches. */
fmm_status fmm_plan_set_graph(fmm_plan* plan, int on);

/* Number of kernels of this library that one fmm_evaluate call on this plan launches (HOST out): permute, P2M, one M2M
 * and one L2L per level below the coarsest level that holds a weak pair (levels above it carry no far field), M2L (when the weak list is not empty; two launches -- leaf level and upper levels -- in the
 * concurrent schedule with the register kernels), P2P, L2P (which also finalizes).  cudaMemset nodes are not counted. */
fmm_status fmm_plan_launches(const fmm_plan* plan, int64_t* h_launches_per_evaluate);

/* Floating-point instructions that ONE translation executes in the kernels selected for (p, dtype) with m2l_variant 0
 * (HOST outputs, any may be NULL): fused multiply-adds, multiplies, adds of the rotate / z-shift / rotate-back operator
 * (App. B) in the factorised form of DESIGN.md section 5 -- geometry, addressing, staging and the sums over equal
 * targets are not counted.  kind: 0 = M2M, 1 = M2L, 2 = L2L.  All zero where only the generic kernels exist (p = 0, p > 12).
 * This is the per-unit work behind bench.py's roofline line: executed flop = 2 * fma + mul + add.  No device needed. */
fmm_status fmm_translation_work(int p, fmm_dtype dtype, int kind, int64_t* h_fma, int64_t* h_mul, int64_t* h_add);

/* Thread-local, NUL-terminated description of the last failure on the calling thread ("" if none). */
const char* fmm_last_error(void);

/* Library version string. */
const char* fmm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PAPER_2511_15269_FMM_H */
