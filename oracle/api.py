"""ctypes front-end of the CPU oracle (oracle/fmm_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs; never by the product package.  Argument marshalling only -- all arithmetic is in
fmm_oracle.cpp, whose functions cite the PAPER.md passages they follow.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)
_bp = C.POINTER(C.c_uint8)


def _d(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _i(a):
    return a.ctypes.data_as(_ip) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_regular_basis.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp]
        L.orc_singular_basis.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp]
        L.orc_regular_grad.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp]
        L.orc_wigner_d.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_wigner_d.restype = C.c_double
        L.orc_rot_azimuthal.argtypes = [C.c_int, C.c_int, _dp, C.c_double, _dp]
        L.orc_rot_polar.argtypes = [C.c_int, C.c_int, _dp, C.c_double, _dp]
        L.orc_shift.argtypes = [C.c_int, C.c_int, _dp, C.c_double, _dp]
        L.orc_translate.argtypes = [C.c_int, C.c_int, _dp, _dp, _dp]
        L.orc_tree_depth.argtypes = [C.c_int64, C.c_int, C.c_int]
        L.orc_tree_depth.restype = C.c_int
        L.orc_plan_create.argtypes = [_dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int]
        L.orc_plan_create.restype = C.c_void_p
        L.orc_plan_destroy.argtypes = [C.c_void_p]
        L.orc_plan_info.argtypes = [C.c_void_p, C.POINTER(C.c_int)] + [_ip] * 5
        L.orc_plan_copy_tree.argtypes = [C.c_void_p, _ip, _ip, _ip, _dp, _dp, _dp, _dp]
        L.orc_plan_copy_lists.argtypes = [C.c_void_p, _ip, _ip, _ip, _ip]
        L.orc_lists_from_geometry.argtypes = [C.c_int, C.c_int, _dp, _dp, C.c_double, C.c_int, _ip, _ip]
        L.orc_evaluate.argtypes = [C.c_void_p, _dp, _bp, _dp, _dp, C.c_int]
        L.orc_evaluate_adjoint.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_int]
        L.orc_direct.argtypes = [_dp, _dp, C.c_int64, _ip, C.c_int64, _dp, _dp, C.c_int]
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        _i32p = C.POINTER(C.c_int)
        L.orc_plan_st_create.argtypes = [_dp, C.c_int64, _dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_plan_st_create.restype = C.c_void_p
        L.orc_plan_st_destroy.argtypes = [C.c_void_p]
        L.orc_plan_st_info.argtypes = [C.c_void_p, C.c_int, _i32p] + [_ip] * 5 + [_i32p]
        L.orc_plan_st_copy_tree.argtypes = [C.c_void_p, C.c_int, _ip, _ip, _ip, _dp, _dp, _dp, _dp]
        L.orc_plan_st_copy_lists.argtypes = [C.c_void_p, _ip, _ip, _ip, _ip, _i32p]
        L.orc_evaluate_st.argtypes = [C.c_void_p, _dp, _bp, _dp, _dp, C.c_int]
        L.orc_evaluate_st_adjoint.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_int]
        L.orc_direct_st.argtypes = [_dp, _dp, C.c_int64, _dp, C.c_int64, _dp, _dp, C.c_int]
        _lib = L
    return _lib


def nk(p):
    return (p + 1) * (p + 1)


def idx(n, m):
    return n * n + n + m


def regular_basis(p, r):
    out = np.empty(nk(p))
    lib().orc_regular_basis(p, float(r[0]), float(r[1]), float(r[2]), _d(out))
    return out


def singular_basis(p, r):
    out = np.empty(nk(p))
    lib().orc_singular_basis(p, float(r[0]), float(r[1]), float(r[2]), _d(out))
    return out


def regular_grad(p, r):
    out = np.empty((nk(p), 3))
    lib().orc_regular_grad(p, float(r[0]), float(r[1]), float(r[2]), _d(out))
    return out


def wigner_d(j, mp, m, beta):
    return lib().orc_wigner_d(j, mp, m, float(beta))


def rot_azimuthal(p, local_type, v, dphi):
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.empty_like(v)
    lib().orc_rot_azimuthal(p, int(local_type), _d(v), float(dphi), _d(out))
    return out


def rot_polar(p, local_type, v, dtheta):
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.empty_like(v)
    lib().orc_rot_polar(p, int(local_type), _d(v), float(dtheta), _d(out))
    return out


M2M, M2L, L2L = 0, 1, 2


def shift(kind, p, v, r):
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.empty_like(v)
    lib().orc_shift(kind, p, _d(v), float(r), _d(out))
    return out


def translate(kind, p, v, b):
    v = np.ascontiguousarray(v, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    out = np.empty_like(v)
    lib().orc_translate(kind, p, _d(v), _d(b), _d(out))
    return out


def tree_depth(N, N_max, s):
    return lib().orc_tree_depth(int(N), int(N_max), int(s))


def num_threads():
    return lib().orc_num_threads()


def set_num_threads(n):
    """OpenMP threads of the following oracle calls (n < 1: all processors).  Timing control only -- results do not depend on it."""
    lib().orc_set_num_threads(int(n))


class Plan:
    """Oracle hierarchy + lists for fixed positions (reusable for new charges)."""

    def __init__(self, pos, p, N_max, s, theta=0.77, cross_level=0):
        self.pos = np.ascontiguousarray(pos, dtype=np.float64)
        assert self.pos.ndim == 2 and self.pos.shape[1] == 3
        self.N = self.pos.shape[0]
        self.p, self.N_max, self.s, self.theta = int(p), int(N_max), int(s), float(theta)
        self.cross_level = int(cross_level)
        self._h = lib().orc_plan_create(_d(self.pos), self.N, self.p, self.N_max, self.s, self.theta, self.cross_level)
        L = C.c_int()
        v = [C.c_int64() for _ in range(5)]
        lib().orc_plan_info(self._h, C.byref(L), *[C.byref(x) for x in v])
        self.L = L.value
        self.n_boxes, self.n_leaves, self.n_weak, self.n_strong, self.n_p2p_pairs = [x.value for x in v]

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_plan_destroy(self._h)
            self._h = None

    def tree(self):
        nb = self.n_boxes
        t = dict(perm=np.empty(self.N, np.int64), box_start=np.empty(nb, np.int64), box_count=np.empty(nb, np.int64),
                 lo=np.empty((nb, 3)), hi=np.empty((nb, 3)), ctr=np.empty((nb, 3)), rad=np.empty(nb))
        lib().orc_plan_copy_tree(self._h, _i(t["perm"]), _i(t["box_start"]), _i(t["box_count"]), _d(t["lo"]), _d(t["hi"]),
                                 _d(t["ctr"]), _d(t["rad"]))
        return t

    def lists(self):
        ls = dict(weak_off=np.empty(self.n_boxes + 1, np.int64), weak_src=np.empty(self.n_weak, np.int64),
                  strong_off=np.empty(self.n_leaves + 1, np.int64), strong_src=np.empty(self.n_strong, np.int64))
        lib().orc_plan_copy_lists(self._h, _i(ls["weak_off"]), _i(ls["weak_src"]), _i(ls["strong_off"]), _i(ls["strong_src"]))
        return ls

    def evaluate(self, q, leaf_mask=None, want_field=True, fp32_rule=False):
        """potential (N,), field (N,3) in input order.  With leaf_mask (n_leaves uint8) only the particles of
        the masked leaves are written; the others are NaN.  fp32_rule: coincidence (reading S3) is decided in binary32,
        as the fp32 CUDA kernels decide it (pairs with r^2 < FLT_MIN are skipped); for comparisons with fp32 plans."""
        q = np.ascontiguousarray(q, dtype=np.float64)
        assert q.shape == (self.N,)
        pot = np.full(self.N, np.nan)
        fld = np.full((self.N, 3), np.nan) if want_field else None
        m = None
        if leaf_mask is not None:
            m = np.ascontiguousarray(leaf_mask, dtype=np.uint8)
            assert m.shape == (self.n_leaves,)
        lib().orc_evaluate(self._h, _d(q), m.ctypes.data_as(_bp) if m is not None else None, _d(pot), _d(fld), int(fp32_rule))
        return pot, fld

    def evaluate_adjoint(self, ubar=None, fbar=None, fp32_rule=False):
        """qbar (N,) = A^T ubar + F^T fbar: the vector-Jacobian product of evaluate() with respect to the charges
        (PAPER.md:281-310), every step transposed.  ubar (N,) and / or fbar (N,3): cotangents of potential and field."""
        ub = None if ubar is None else np.ascontiguousarray(ubar, dtype=np.float64)
        fb = None if fbar is None else np.ascontiguousarray(fbar, dtype=np.float64)
        assert ub is None or ub.shape == (self.N,)
        assert fb is None or fb.shape == (self.N, 3)
        qbar = np.empty(self.N)
        lib().orc_evaluate_adjoint(self._h, _d(ub), _d(fb), _d(qbar), int(fp32_rule))
        return qbar


def lists_from_geometry(s, L, ctr, rad, theta, cross_level=0):
    ctr = np.ascontiguousarray(ctr, dtype=np.float64)
    rad = np.ascontiguousarray(rad, dtype=np.float64)
    nb = rad.shape[0]
    nw = np.empty(nb, np.int64)
    ns = np.empty(1 << (s * L), np.int64)
    lib().orc_lists_from_geometry(s, L, _d(ctr), _d(rad), float(theta), int(cross_level), _i(nw), _i(ns))
    return nw, ns


def direct(pos, q, targets=None, fp32_rule=False):
    """Plain definition eqs. (1)-(3): u_i = -(1/4pi) sum_{j!=i} q_j/|r_i-r_j|, field = -grad u, at `targets`."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64)
    N = pos.shape[0]
    tg = np.arange(N, dtype=np.int64) if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    pot = np.empty(tg.shape[0])
    fld = np.empty((tg.shape[0], 3))
    lib().orc_direct(_d(pos), _d(q), N, _i(tg), tg.shape[0], _d(pot), _d(fld), int(fp32_rule))
    return pot, fld


class PlanST:
    """Oracle plan for separate sources and targets: two hierarchies, level-marching lists."""

    def __init__(self, src_pos, tgt_pos, p, N_max, s, theta=0.77):
        self.spos = np.ascontiguousarray(src_pos, dtype=np.float64)
        self.tpos = np.ascontiguousarray(tgt_pos, dtype=np.float64)
        assert self.spos.ndim == 2 and self.spos.shape[1] == 3 and self.tpos.ndim == 2 and self.tpos.shape[1] == 3
        self.Ns, self.Nt = self.spos.shape[0], self.tpos.shape[0]
        self.p, self.N_max, self.s, self.theta = int(p), int(N_max), int(s), float(theta)
        self._h = lib().orc_plan_st_create(_d(self.spos), self.Ns, _d(self.tpos), self.Nt, self.p, self.N_max, self.s, self.theta)
        self.info = {}
        for which, name in ((0, "src"), (1, "tgt")):
            L = C.c_int()
            ns = C.c_int()
            v = [C.c_int64() for _ in range(5)]
            lib().orc_plan_st_info(self._h, which, C.byref(L), *[C.byref(x) for x in v], C.byref(ns))
            self.info[name] = dict(L=L.value, n_boxes=v[0].value, n_leaves=v[1].value)
            self.n_weak, self.n_strong, self.n_p2p_pairs, self.n_steps = v[2].value, v[3].value, v[4].value, ns.value

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_plan_st_destroy(self._h)
            self._h = None

    def tree(self, which):
        """which: 'src' or 'tgt'"""
        w = 0 if which == "src" else 1
        nb = self.info[which]["n_boxes"]
        N = self.Ns if w == 0 else self.Nt
        t = dict(perm=np.empty(N, np.int64), box_start=np.empty(nb, np.int64), box_count=np.empty(nb, np.int64),
                 lo=np.empty((nb, 3)), hi=np.empty((nb, 3)), ctr=np.empty((nb, 3)), rad=np.empty(nb))
        lib().orc_plan_st_copy_tree(self._h, w, _i(t["perm"]), _i(t["box_start"]), _i(t["box_count"]), _d(t["lo"]), _d(t["hi"]),
                                    _d(t["ctr"]), _d(t["rad"]))
        return t

    def lists(self):
        """weak: CSR by target box (global id in the target hierarchy), sources = global ids in the source hierarchy;
        strong: CSR by target leaf, sources = source leaf indices; steps: the (l_trg, l_src) pairs visited."""
        ls = dict(weak_off=np.empty(self.info["tgt"]["n_boxes"] + 1, np.int64), weak_src=np.empty(self.n_weak, np.int64),
                  strong_off=np.empty(self.info["tgt"]["n_leaves"] + 1, np.int64), strong_src=np.empty(self.n_strong, np.int64))
        steps = np.empty(2 * self.n_steps, np.int32)
        lib().orc_plan_st_copy_lists(self._h, _i(ls["weak_off"]), _i(ls["weak_src"]), _i(ls["strong_off"]), _i(ls["strong_src"]),
                                     steps.ctypes.data_as(C.POINTER(C.c_int)))
        ls["steps"] = steps.reshape(-1, 2)
        return ls

    def evaluate(self, q, leaf_mask=None, fp32_rule=False):
        """potential (Nt,), field (Nt,3) at the targets, in target input order.  With leaf_mask (uint8 per target leaf) only
        the targets of the masked leaves are written; the others are NaN."""
        q = np.ascontiguousarray(q, dtype=np.float64)
        assert q.shape == (self.Ns,)
        pot = np.full(self.Nt, np.nan)
        fld = np.full((self.Nt, 3), np.nan)
        m = None
        if leaf_mask is not None:
            m = np.ascontiguousarray(leaf_mask, dtype=np.uint8)
            assert m.shape == (self.info["tgt"]["n_leaves"],)
        lib().orc_evaluate_st(self._h, _d(q), m.ctypes.data_as(_bp) if m is not None else None, _d(pot), _d(fld), int(fp32_rule))
        return pot, fld

    def evaluate_adjoint(self, ubar=None, fbar=None, fp32_rule=False):
        """qbar (Ns,) = A^T ubar + F^T fbar for cotangents ubar (Nt,), fbar (Nt,3) of the outputs of evaluate()."""
        ub = None if ubar is None else np.ascontiguousarray(ubar, dtype=np.float64)
        fb = None if fbar is None else np.ascontiguousarray(fbar, dtype=np.float64)
        assert ub is None or ub.shape == (self.Nt,)
        assert fb is None or fb.shape == (self.Nt, 3)
        qbar = np.empty(self.Ns)
        lib().orc_evaluate_st_adjoint(self._h, _d(ub), _d(fb), _d(qbar), int(fp32_rule))
        return qbar


def direct_st(src_pos, q, tgt_pos, fp32_rule=False):
    """Plain definition at separate targets: u(t_i) = -(1/4pi) sum_j q_j/|t_i - s_j|, field = -grad u."""
    sp = np.ascontiguousarray(src_pos, dtype=np.float64)
    tp = np.ascontiguousarray(tgt_pos, dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64)
    pot = np.empty(tp.shape[0])
    fld = np.empty((tp.shape[0], 3))
    lib().orc_direct_st(_d(sp), _d(q), sp.shape[0], _d(tp), tp.shape[0], _d(pot), _d(fld), int(fp32_rule))
    return pot, fld
