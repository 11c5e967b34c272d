"""Thin Python binding of include/fmm.h (argument marshalling only; every step runs in the CUDA library).

Loads the in-tree library paper_2511_15269_b200/libfmm_b200.so and FAILS LOUDLY if it is missing -- there
is no CPU or PyTorch fallback.  PyTorch is used only for device memory (tensor.data_ptr()) and streams.
Function names mirror the C entry points; `Plan` is a small convenience wrapper around them.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfmm_b200.so")

FMM_OK, FMM_ERR_INVALID_ARG, FMM_ERR_ALLOC, FMM_ERR_CUDA, FMM_ERR_UNSUPPORTED = 0, 1, 2, 3, 4
FMM_F32, FMM_F64 = 0, 1
FMM_P_MAX = 16

EXPORTS = ["fmm_plan_create", "fmm_evaluate", "fmm_evaluate_adjoint", "fmm_evaluate_host", "fmm_evaluate_host_submit", "fmm_evaluate_host_wait", "fmm_plan_destroy", "fmm_plan_info", "fmm_plan_copy_tree",
           "fmm_plan_copy_lists", "fmm_evaluate_profiled", "fmm_plan_timings", "fmm_plan_set_m2l_variant", "fmm_plan_set_deterministic", "fmm_plan_set_schedule", "fmm_plan_set_graph", "fmm_plan_launches", "fmm_last_error",
           "fmm_version", "fmm_translation_work", "fmm_plan_update", "fmm_shard_box_range", "fmm_evaluate_shard_upward",
           "fmm_evaluate_shard_downward", "fmm_plan_leaf_multipoles", "fmm_leaf_multipoles_noalloc", "fmm_plan_create_targets", "fmm_plan_source_info", "fmm_plan_copy_source_tree", "fmm_plan_copy_march"]


class fmm_admissibility(C.Structure):
    _fields_ = [("theta", C.c_double), ("cross_level", C.c_int)]


class FmmError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("fmm status %d: %s" % (status, msg))
        self.status = status


_lib = None


def lib():
    """The loaded C-ABI library.  Raises ImportError if the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("CUDA library %s is missing: run `python -m paper_2511_15269_b200.build` (no fallback exists)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, i64p, i32p, dp = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32), C.POINTER(C.c_double)
        L.fmm_plan_create.argtypes = [vp, C.c_int64, C.c_int, C.c_int, C.c_int, C.POINTER(fmm_admissibility), C.c_int, vp, C.POINTER(vp)]
        L.fmm_evaluate.argtypes = [vp, vp, vp, vp, vp]
        L.fmm_evaluate_host.argtypes = [vp, vp, vp, vp, vp]
        L.fmm_evaluate_host_submit.argtypes = [vp, vp, vp, vp, vp]
        L.fmm_evaluate_host_wait.argtypes = [vp]
        L.fmm_evaluate_adjoint.argtypes = [vp, vp, vp, vp, vp]
        L.fmm_evaluate_profiled.argtypes = [vp, vp, vp, vp, vp, dp]
        L.fmm_plan_destroy.argtypes = [vp]
        L.fmm_plan_info.argtypes = [vp, C.POINTER(C.c_int), i64p, i64p, i64p, i64p, i64p]
        L.fmm_plan_copy_tree.argtypes = [vp, i32p, i32p, i32p, vp, vp, dp, dp]
        L.fmm_plan_copy_lists.argtypes = [vp, i64p, i32p, i64p, i32p]
        L.fmm_plan_create_targets.argtypes = [vp, C.c_int64, vp, C.c_int64, C.c_int, C.c_int, C.c_int, C.POINTER(fmm_admissibility), C.c_int, vp, C.POINTER(vp)]
        L.fmm_plan_update.argtypes = [vp, vp, vp, vp]
        L.fmm_shard_box_range.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, i64p, i64p]
        L.fmm_evaluate_shard_upward.argtypes = [vp, C.c_int, C.c_int, vp, vp]
        L.fmm_evaluate_shard_downward.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp]
        L.fmm_plan_leaf_multipoles.argtypes = [vp, C.c_int, C.c_int64, C.c_int64, vp, i64p, vp]
        L.fmm_leaf_multipoles_noalloc.argtypes = [vp, vp, vp, i64p, vp]
        L.fmm_plan_source_info.argtypes = [vp, i64p, C.POINTER(C.c_int), i64p, i64p]
        L.fmm_plan_copy_source_tree.argtypes = [vp, i32p, i32p, i32p, vp, vp, dp, dp]
        L.fmm_plan_copy_march.argtypes = [vp, i32p, i32p]
        L.fmm_plan_timings.argtypes = [vp, dp]
        L.fmm_plan_set_m2l_variant.argtypes = [vp, C.c_int]
        L.fmm_plan_set_deterministic.argtypes = [vp, C.c_int, vp]
        L.fmm_plan_set_schedule.argtypes = [vp, C.c_int]
        L.fmm_plan_set_graph.argtypes = [vp, C.c_int]
        L.fmm_plan_launches.argtypes = [vp, i64p]
        L.fmm_translation_work.argtypes = [C.c_int, C.c_int, C.c_int, i64p, i64p, i64p]
        L.fmm_last_error.restype = C.c_char_p
        L.fmm_version.restype = C.c_char_p
        for name in EXPORTS:
            if getattr(L, name).restype is C.c_int:
                pass
        _lib = L
    return _lib


def fmm_last_error():
    return lib().fmm_last_error().decode()


def fmm_version():
    return lib().fmm_version().decode()


def _check(st):
    if st != FMM_OK:
        raise FmmError(st, fmm_last_error())


def _dtype_code(t):
    import torch
    if t.dtype == torch.float32:
        return FMM_F32
    if t.dtype == torch.float64:
        return FMM_F64
    raise TypeError("positions/charges must be float32 or float64")


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


# handle -> (torch dtype, number of charges, number of outputs, device): the C side sees raw pointers only, so the binding checks
# every tensor it marshals against the plan it is passed with
_PLANS = {}


def _check_io(plan, charges, potential, field, host=False):
    meta = _PLANS.get(plan.value)
    if meta is None:
        raise ValueError("unknown or destroyed plan handle")
    tdtype, Nq, Nt, device = meta

    def one(name, t, shape):
        if t is None:
            return
        if isinstance(t, np.ndarray):
            if not host:
                raise ValueError("%s must be a CUDA tensor" % name)
            ok_dtype = t.dtype == (np.float32 if str(tdtype).endswith("float32") else np.float64)
            contiguous, on_dev = t.flags["C_CONTIGUOUS"], True
        else:
            ok_dtype = t.dtype == tdtype
            contiguous = t.is_contiguous()
            on_dev = (not t.is_cuda) if host else (t.is_cuda and t.device == device)
        if not ok_dtype:
            raise ValueError("%s has dtype %s but the plan was built for %s" % (name, t.dtype, tdtype))
        if tuple(t.shape) != shape:
            raise ValueError("%s has shape %s, expected %s" % (name, tuple(t.shape), shape))
        if not contiguous:
            raise ValueError("%s must be contiguous" % name)
        if not on_dev:
            raise ValueError("%s must live %s" % (name, "in host memory" if host else "on the plan's device %s" % device))

    one("charges", charges, (Nq,))
    one("potential", potential, (Nt,))
    one("field", field, (Nt, 3))


def fmm_plan_create(positions, p, N_max, s, theta=0.77, cross_level=0, stream=None):
    """positions: CUDA tensor (N,3), contiguous, float32/float64.  Returns an opaque plan handle (c_void_p)."""
    if not positions.is_cuda or not positions.is_contiguous() or positions.dim() != 2 or positions.shape[1] != 3:
        raise ValueError("positions must be a contiguous CUDA tensor of shape (N,3)")
    adm = fmm_admissibility(float(theta), int(cross_level))
    h = C.c_void_p()
    _check(lib().fmm_plan_create(C.c_void_p(positions.data_ptr()), positions.shape[0], int(p), int(N_max), int(s), C.byref(adm),
                                 _dtype_code(positions), _stream_ptr(stream), C.byref(h)))
    _PLANS[h.value] = (positions.dtype, positions.shape[0], positions.shape[0], positions.device)
    return h


def fmm_plan_create_targets(sources, targets, p, N_max, s, theta=0.77, stream=None):
    """sources (Ns,3), targets (Nt,3): contiguous CUDA tensors of one dtype.  Returns a plan handle."""
    for a in (sources, targets):
        if not a.is_cuda or not a.is_contiguous() or a.dim() != 2 or a.shape[1] != 3:
            raise ValueError("sources and targets must be contiguous CUDA tensors of shape (N,3)")
    if sources.dtype != targets.dtype:
        raise ValueError("sources and targets must have the same dtype")
    adm = fmm_admissibility(float(theta), 1)
    h = C.c_void_p()
    _check(lib().fmm_plan_create_targets(C.c_void_p(sources.data_ptr()), sources.shape[0], C.c_void_p(targets.data_ptr()), targets.shape[0], int(p),
                                         int(N_max), int(s), C.byref(adm), _dtype_code(sources), _stream_ptr(stream), C.byref(h)))
    _PLANS[h.value] = (sources.dtype, sources.shape[0], targets.shape[0], sources.device)
    return h


def fmm_plan_update(plan, positions=None, targets=None, stream=None):
    """Re-plan in place for moved points (same counts, dtype and parameters).  One point set: `positions`; separate targets:
    `positions` = new sources and / or `targets` = new targets (None = unchanged)."""
    meta = _PLANS.get(plan.value)
    if meta is None:
        raise ValueError("unknown or destroyed plan handle")
    tdtype, Nq, Nt, device = meta
    for t, n in ((positions, Nq), (targets, Nt)):
        if t is not None and (not t.is_cuda or not t.is_contiguous() or t.dtype != tdtype or tuple(t.shape) != (n, 3) or t.device != device):
            raise ValueError("new positions must be contiguous CUDA tensors of shape (%d, 3) and dtype %s on %s" % (n, tdtype, device))
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(lib().fmm_plan_update(plan, p(positions), p(targets), _stream_ptr(stream)))


def fmm_shard_box_range(L, s, n_shards, shard, level):
    """level-local [begin, end) of the boxes of `level` that shard `shard` of `n_shards` touches (no device needed)"""
    a, b = C.c_int64(), C.c_int64()
    _check(lib().fmm_shard_box_range(int(L), int(s), int(n_shards), int(shard), int(level), C.byref(a), C.byref(b)))
    return a.value, b.value


def fmm_evaluate_shard_upward(plan, n_shards, shard, charges, stream=None):
    _check_io(plan, charges, None, None)
    _check(lib().fmm_evaluate_shard_upward(plan, int(n_shards), int(shard), C.c_void_p(charges.data_ptr()), _stream_ptr(stream)))


def fmm_evaluate_shard_downward(plan, n_shards, shard, potential=None, field=None, stream=None):
    _check_io(plan, None, potential, field)
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(lib().fmm_evaluate_shard_downward(plan, int(n_shards), int(shard), p(potential), p(field), _stream_ptr(stream)))


def fmm_plan_leaf_multipoles(plan, copy_in, leaf_begin, leaf_end, rows=None, stream=None):
    """copies leaf rows of the multipole array out of (copy_in = 0) or into (1) the plan; returns the row length in elements"""
    n = C.c_int64()
    _check(lib().fmm_plan_leaf_multipoles(plan, int(copy_in), int(leaf_begin), int(leaf_end), C.c_void_p(rows.data_ptr()) if rows is not None else None,
                                          C.byref(n), _stream_ptr(stream)))
    return n.value


FMM_NOALLOC_MAX_BYTES = 8 << 20


def fmm_leaf_multipoles_noalloc(plan, charges=None, rows=None, stream=None):
    """P2M of all leaves for `charges` (N,) into `rows` (n_leaves, row): no allocation, scratch in a static device array of
    FMM_NOALLOC_MAX_BYTES (N <= 524288 fp32 / 262144 fp64), nothing of the plan is written; see include/fmm.h.  Returns the row
    length in elements; charges = rows = None only queries it."""
    n = C.c_int64()
    if charges is not None:
        _check_io(plan, charges, None, None)
    if rows is not None:
        meta = _PLANS.get(plan.value)
        if meta is None or rows.dtype != meta[0] or not rows.is_cuda or not rows.is_contiguous() or rows.device != meta[3]:
            raise ValueError("rows must be a contiguous CUDA tensor of the plan's dtype on the plan's device")
    _check(lib().fmm_leaf_multipoles_noalloc(plan, C.c_void_p(charges.data_ptr()) if charges is not None else None,
                                             C.c_void_p(rows.data_ptr()) if rows is not None else None, C.byref(n), _stream_ptr(stream)))
    return n.value


def evaluate_sharded(plan, n_leaves, charges, potential=None, field=None, group=None):
    """One evaluate with the targets sharded over the ranks of a torch.distributed process group (one process per GPU; every rank
    holds the same plan and all charges): upward pass for the own leaves, ONE all-gather of the leaf multipoles (NCCL over NVLink
    on GPUs), downward pass for the own targets.  Writes the potential / field of the own particles only."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    fmm_evaluate_shard_upward(plan, world, rank, charges)
    if world > 1:
        kp = fmm_plan_leaf_multipoles(plan, 0, 0, 0)
        bounds = [n_leaves * r // world for r in range(world + 1)]
        rows = max(b - a for a, b in zip(bounds, bounds[1:]))
        mine = torch.zeros((rows, kp), dtype=charges.dtype, device=charges.device)
        fmm_plan_leaf_multipoles(plan, 0, bounds[rank], bounds[rank + 1], mine)
        allrows = torch.empty((world, rows, kp), dtype=charges.dtype, device=charges.device)
        dist.all_gather_into_tensor(allrows, mine, group=group)
        for r in range(world):
            if r != rank and bounds[r + 1] > bounds[r]:
                fmm_plan_leaf_multipoles(plan, 1, bounds[r], bounds[r + 1], allrows[r])
    fmm_evaluate_shard_downward(plan, world, rank, potential, field)


def fmm_plan_source_info(plan):
    Ns, L, nb, nl = C.c_int64(), C.c_int(), C.c_int64(), C.c_int64()
    _check(lib().fmm_plan_source_info(plan, C.byref(Ns), C.byref(L), C.byref(nb), C.byref(nl)))
    return dict(N=Ns.value, L=L.value, n_boxes=nb.value, n_leaves=nl.value)


def fmm_plan_copy_source_tree(plan, dtype):
    info = fmm_plan_source_info(plan)
    nb, N = info["n_boxes"], info["N"]
    fl = np.float32 if dtype == FMM_F32 else np.float64
    t = dict(perm=np.empty(N, np.int32), box_start=np.empty(nb, np.int32), box_count=np.empty(nb, np.int32), lo=np.empty((nb, 3), fl),
             hi=np.empty((nb, 3), fl), ctr=np.empty((nb, 3), np.float64), rad=np.empty(nb, np.float64))
    i32p, dp = C.POINTER(C.c_int32), C.POINTER(C.c_double)
    _check(lib().fmm_plan_copy_source_tree(plan, t["perm"].ctypes.data_as(i32p), t["box_start"].ctypes.data_as(i32p), t["box_count"].ctypes.data_as(i32p),
                                           C.c_void_p(t["lo"].ctypes.data), C.c_void_p(t["hi"].ctypes.data), t["ctr"].ctypes.data_as(dp),
                                           t["rad"].ctypes.data_as(dp)))
    return t


def fmm_plan_copy_march(plan):
    n = C.c_int32()
    _check(lib().fmm_plan_copy_march(plan, None, C.byref(n)))
    steps = np.empty(2 * n.value, np.int32)
    if n.value:
        _check(lib().fmm_plan_copy_march(plan, steps.ctypes.data_as(C.POINTER(C.c_int32)), C.byref(n)))
    return steps.reshape(-1, 2)


def fmm_plan_destroy(plan):
    _PLANS.pop(plan.value, None)
    _check(lib().fmm_plan_destroy(plan))


def fmm_evaluate(plan, charges, potential=None, field=None, stream=None):
    """charges (N,), potential (N,) or None, field (N,3) or None: contiguous CUDA tensors of the plan's dtype on the plan's device
    (N = number of sources for the charges, number of targets for the outputs)."""
    _check_io(plan, charges, potential, field)
    _check(lib().fmm_evaluate(plan, C.c_void_p(charges.data_ptr()), C.c_void_p(potential.data_ptr()) if potential is not None else None,
                              C.c_void_p(field.data_ptr()) if field is not None else None, _stream_ptr(stream)))


def fmm_evaluate_adjoint(plan, cot_potential, cot_field, charge_grad, stream=None):
    """charge_grad (Ns,) = A^T cot_potential + F^T cot_field: the VJP of fmm_evaluate with respect to the charges.
    cot_potential (Nt,) and / or cot_field (Nt,3): contiguous CUDA tensors of the plan's dtype; one of them may be None."""
    if cot_potential is None and cot_field is None:
        raise ValueError("at least one cotangent is needed")
    _check_io(plan, charge_grad, cot_potential, cot_field)
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(lib().fmm_evaluate_adjoint(plan, p(cot_potential), p(cot_field), p(charge_grad), _stream_ptr(stream)))


def fmm_evaluate_profiled(plan, charges, potential=None, field=None, stream=None):
    _check_io(plan, charges, potential, field)
    ms = (C.c_double * 8)()
    _check(lib().fmm_evaluate_profiled(plan, C.c_void_p(charges.data_ptr()), C.c_void_p(potential.data_ptr()) if potential is not None else None,
                                       C.c_void_p(field.data_ptr()) if field is not None else None, _stream_ptr(stream), ms))
    names = ["permute", "p2m", "m2m", "m2l", "l2l", "l2p", "p2p", "total"]
    return dict(zip(names, list(ms)))


def fmm_evaluate_host(plan, h_charges, h_potential=None, h_field=None, stream=None):
    """Host-buffer path: numpy arrays or pinned CPU tensors; H2D and D2H copies happen inside the call."""
    _check_io(plan, h_charges, h_potential, h_field, host=True)

    def ptr(a):
        if a is None:
            return None
        if isinstance(a, np.ndarray):
            return C.c_void_p(a.ctypes.data)
        return C.c_void_p(a.data_ptr())
    _check(lib().fmm_evaluate_host(plan, ptr(h_charges), ptr(h_potential), ptr(h_field), _stream_ptr(stream)))


def _host_ptr(a):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return C.c_void_p(a.ctypes.data)
    return C.c_void_p(a.data_ptr())


def fmm_evaluate_host_submit(plan, h_charges, h_potential=None, h_field=None, stream=None):
    """Pipelined host path: enqueue H2D + evaluate + D2H and return; at most two calls in flight (pinned buffers to overlap)."""
    _check_io(plan, h_charges, h_potential, h_field, host=True)
    _check(lib().fmm_evaluate_host_submit(plan, _host_ptr(h_charges), _host_ptr(h_potential), _host_ptr(h_field), _stream_ptr(stream)))


def fmm_evaluate_host_wait(plan):
    """Block until the oldest submitted call has written its results into its host buffers."""
    _check(lib().fmm_evaluate_host_wait(plan))


def fmm_plan_info(plan):
    L = C.c_int()
    v = [C.c_int64() for _ in range(5)]
    _check(lib().fmm_plan_info(plan, C.byref(L), *[C.byref(x) for x in v]))
    return dict(L=L.value, n_boxes=v[0].value, n_leaves=v[1].value, n_weak=v[2].value, n_strong=v[3].value, n_p2p_pairs=v[4].value)


def fmm_plan_timings(plan):
    ms = (C.c_double * 4)()
    _check(lib().fmm_plan_timings(plan, ms))
    return dict(sort=ms[0], tree=ms[1], lists=ms[2], total=ms[3])


def fmm_plan_launches(plan):
    v = C.c_int64()
    _check(lib().fmm_plan_launches(plan, C.byref(v)))
    return v.value


def fmm_translation_work(p, dtype, kind):
    """(fma, mul, add) instructions of one translation (kind 0 = M2M, 1 = M2L, 2 = L2L) in the specialised kernels."""
    a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().fmm_translation_work(int(p), int(dtype), int(kind), C.byref(a), C.byref(b), C.byref(c)))
    return a.value, b.value, c.value


def fmm_plan_set_schedule(plan, serial):
    _check(lib().fmm_plan_set_schedule(plan, int(serial)))


def fmm_plan_set_graph(plan, on):
    """0 never / 1 always / 2 (default) below 2^19 points: repeated evaluates with the same device pointers replay a captured CUDA graph"""
    _check(lib().fmm_plan_set_graph(plan, int(on)))


def fmm_plan_set_deterministic(plan, on, stream=None):
    """on = 1: bit-for-bit reproducible evaluates (ordered sums, serial schedule); see include/fmm.h"""
    _check(lib().fmm_plan_set_deterministic(plan, int(on), _stream_ptr(stream)))


def fmm_plan_set_m2l_variant(plan, variant):
    _check(lib().fmm_plan_set_m2l_variant(plan, int(variant)))


def fmm_plan_copy_tree(plan, N, dtype):
    info = fmm_plan_info(plan)
    nb = info["n_boxes"]
    fl = np.float32 if dtype == FMM_F32 else np.float64
    t = dict(perm=np.empty(N, np.int32), box_start=np.empty(nb, np.int32), box_count=np.empty(nb, np.int32), lo=np.empty((nb, 3), fl),
             hi=np.empty((nb, 3), fl), ctr=np.empty((nb, 3), np.float64), rad=np.empty(nb, np.float64))
    i32p, dp = C.POINTER(C.c_int32), C.POINTER(C.c_double)
    _check(lib().fmm_plan_copy_tree(plan, t["perm"].ctypes.data_as(i32p), t["box_start"].ctypes.data_as(i32p), t["box_count"].ctypes.data_as(i32p),
                                    C.c_void_p(t["lo"].ctypes.data), C.c_void_p(t["hi"].ctypes.data), t["ctr"].ctypes.data_as(dp),
                                    t["rad"].ctypes.data_as(dp)))
    return t


def fmm_plan_copy_lists(plan):
    info = fmm_plan_info(plan)
    ls = dict(weak_off=np.empty(info["n_boxes"] + 1, np.int64), weak_src=np.empty(info["n_weak"], np.int32),
              strong_off=np.empty(info["n_leaves"] + 1, np.int64), strong_src=np.empty(info["n_strong"], np.int32))
    i32p, i64p = C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    _check(lib().fmm_plan_copy_lists(plan, ls["weak_off"].ctypes.data_as(i64p), ls["weak_src"].ctypes.data_as(i32p),
                                     ls["strong_off"].ctypes.data_as(i64p), ls["strong_src"].ctypes.data_as(i32p)))
    return ls


class Plan:
    """gen_hierarchy(...) / eval_potential(...) of Listing 1 as an object: build once, evaluate many."""

    def __init__(self, positions, p, N_max, s, theta=0.77, stream=None, cross_level=0):
        self.N = positions.shape[0]
        self.dtype = _dtype_code(positions)
        self.tdtype = positions.dtype
        self.device = positions.device
        self.p, self.N_max, self.s, self.theta = p, N_max, s, theta
        self.cross_level = int(cross_level)
        self.handle = fmm_plan_create(positions, p, N_max, s, theta, self.cross_level, stream)
        self.info = fmm_plan_info(self.handle)

    def evaluate(self, charges, want_potential=True, want_field=True, stream=None):
        import torch
        pot = torch.empty(self.N, dtype=self.tdtype, device=self.device) if want_potential else None
        fld = torch.empty((self.N, 3), dtype=self.tdtype, device=self.device) if want_field else None
        fmm_evaluate(self.handle, charges, pot, fld, stream)
        return pot, fld

    def update(self, positions, stream=None):
        """re-plan in place for moved points (fmm_plan_update)"""
        fmm_plan_update(self.handle, positions, None, stream)
        self.info = fmm_plan_info(self.handle)

    def evaluate_adjoint(self, cot_potential=None, cot_field=None, stream=None):
        """gradient of <cot_potential, potential> + <cot_field, field> with respect to the charges (N,)"""
        import torch
        g = torch.empty(self.N, dtype=self.tdtype, device=self.device)
        fmm_evaluate_adjoint(self.handle, cot_potential, cot_field, g, stream)
        return g

    def tree(self):
        return fmm_plan_copy_tree(self.handle, self.N, self.dtype)

    def lists(self):
        return fmm_plan_copy_lists(self.handle)

    def timings(self):
        return fmm_plan_timings(self.handle)

    def close(self):
        if self.handle is not None:
            fmm_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class PlanTargets:
    """Separate sources and targets: potential / field at `targets` from charges at `sources`."""

    def __init__(self, sources, targets, p, N_max, s, theta=0.77, stream=None):
        self.Ns, self.Nt = sources.shape[0], targets.shape[0]
        self.dtype = _dtype_code(sources)
        self.tdtype = sources.dtype
        self.device = sources.device
        self.p, self.N_max, self.s, self.theta = p, N_max, s, theta
        self.handle = fmm_plan_create_targets(sources, targets, p, N_max, s, theta, stream)
        self.info = fmm_plan_info(self.handle)
        self.source_info = fmm_plan_source_info(self.handle)

    def evaluate(self, charges, want_potential=True, want_field=True, stream=None):
        import torch
        pot = torch.empty(self.Nt, dtype=self.tdtype, device=self.device) if want_potential else None
        fld = torch.empty((self.Nt, 3), dtype=self.tdtype, device=self.device) if want_field else None
        fmm_evaluate(self.handle, charges, pot, fld, stream)
        return pot, fld

    def update(self, sources=None, targets=None, stream=None):
        """re-plan in place for moved sources and / or targets (fmm_plan_update)"""
        fmm_plan_update(self.handle, sources, targets, stream)
        self.info = fmm_plan_info(self.handle)
        self.source_info = fmm_plan_source_info(self.handle)

    def evaluate_adjoint(self, cot_potential=None, cot_field=None, stream=None):
        """gradient of <cot_potential, potential> + <cot_field, field> with respect to the source charges (Ns,)"""
        import torch
        g = torch.empty(self.Ns, dtype=self.tdtype, device=self.device)
        fmm_evaluate_adjoint(self.handle, cot_potential, cot_field, g, stream)
        return g

    def tree(self, which):
        """which: 'tgt' or 'src'"""
        return fmm_plan_copy_tree(self.handle, self.Nt, self.dtype) if which == "tgt" else fmm_plan_copy_source_tree(self.handle, self.dtype)

    def lists(self):
        ls = fmm_plan_copy_lists(self.handle)
        ls["steps"] = fmm_plan_copy_march(self.handle)
        return ls

    def timings(self):
        return fmm_plan_timings(self.handle)

    def close(self):
        if self.handle is not None:
            fmm_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
