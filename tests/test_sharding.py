"""Target-sharded evaluate (the paper has no multi-device support).

CPU (`-m "not gpu"`): the partition logic of fmm_shard_box_range -- the leaf ranges of the shards tile the leaf level, the ranges
above are exactly the ancestors -- and a world_size-2 gloo run in which every rank evaluates the ORACLE on the leaves the library
assigns to it (leaf mask) and the results are combined with one collective: the union must equal the full evaluate bit for bit.
GPU: the shards of one evaluate run one after the other on one device (no rank waits for another) and through the leaf-row
exchange of two plans standing in for two ranks; results against the oracle and against the unsharded evaluate."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("L,s", [(0, 3), (1, 1), (3, 2), (5, 3), (13, 1), (4, 3)])
@pytest.mark.parametrize("n", [1, 2, 3, 8, 5])
def test_shard_ranges_tile_the_leaves_and_cover_exactly_the_ancestors(L, s, n):
    nl = 1 << (s * L)
    leaves = [fmm.fmm_shard_box_range(L, s, n, r, L) for r in range(n)]
    assert leaves[0][0] == 0 and leaves[-1][1] == nl
    assert all(a[1] == b[0] for a, b in zip(leaves, leaves[1:]))                      # contiguous, disjoint, complete
    sizes = [b - a for a, b in leaves]
    assert max(sizes) - min(sizes) <= 1                                              # balanced
    for r in range(n):
        lo, hi = leaves[r]
        for level in range(L + 1):
            b0, b1 = fmm.fmm_shard_box_range(L, s, n, r, level)
            anc = sorted({leaf >> (s * (L - level)) for leaf in range(lo, hi)})
            assert list(range(b0, b1)) == anc                                         # exactly the ancestors, as one contiguous range


WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from oracle import api as O
from paper_2511_15269_b200 import fmm, inputs
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["MASTER_PORT"], rank=rank, world_size=world)
pos, q = inputs.uniform_cube(3000, 301)
P = O.Plan(pos, 5, 16, 2, 0.77)
lo, hi = fmm.fmm_shard_box_range(P.L, 2, world, rank, P.L)
mask = np.zeros(P.n_leaves, np.uint8); mask[lo:hi] = 1
u, f = P.evaluate(q, leaf_mask=mask)                       # this rank's targets only (NaN elsewhere)
mine = np.isfinite(u)
buf = torch.from_numpy(np.concatenate([np.where(mine, u, 0.0), np.where(mine[:, None], f, 0.0).ravel(), mine.astype(np.float64)]))
dist.all_reduce(buf)                                       # the collective that assembles the result on every rank
full_u, full_f = P.evaluate(q)
got_u, got_f, cover = buf[:3000].numpy(), buf[3000:12000].numpy().reshape(3000, 3), buf[12000:].numpy()
ok = bool(np.array_equal(got_u, full_u) and np.array_equal(got_f, full_f) and np.all(cover == 1.0))
# weak pairs per shard and level: the leaf-level pieces tile the leaf-level list, upper levels may be shared (redundant work)
ls = P.lists(); off = [sum(4 ** k for k in range(l)) for l in range(P.L + 2)]
pairs = [int(ls["weak_off"][off[l] + fmm.fmm_shard_box_range(P.L, 2, world, rank, l)[1]] - ls["weak_off"][off[l] + fmm.fmm_shard_box_range(P.L, 2, world, rank, l)[0]]) for l in range(P.L + 1)]
print("RESULT " + json.dumps(dict(rank=rank, ok=ok, n_mine=int(mine.sum()), pairs=pairs, leaf_pairs_total=int(ls["weak_off"][off[P.L + 1]] - ls["weak_off"][off[P.L]]))), flush=True)
dist.destroy_process_group()
""" % ROOT


def test_two_gloo_ranks_shard_the_targets_and_reassemble_the_full_result(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = 31500 + os.getpid() % 2000
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    res = {}
    for pr in procs:
        so, se = pr.communicate(timeout=300)
        assert pr.returncode == 0, se[-2000:]
        d = json.loads([l for l in so.splitlines() if l.startswith("RESULT ")][0][7:])
        res[d["rank"]] = d
    assert res[0]["ok"] and res[1]["ok"]
    assert res[0]["n_mine"] + res[1]["n_mine"] == 3000
    assert res[0]["pairs"][-1] + res[1]["pairs"][-1] == res[0]["leaf_pairs_total"]  # the leaf-level M2L work is split, not duplicated


# ------------------------------------------------------------------------------------------------ device
torch = pytest.importorskip("torch")


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel2(a, b):
    return np.linalg.norm(np.asarray(a, np.float64) - b) / np.linalg.norm(b)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,N,N_max,s,p,cross", [(np.float32, 20000, 32, 3, 8, 0), (np.float64, 6000, 16, 2, 6, 1), (np.float32, 5000, 40, 1, 5, 0),
                                                      (np.float64, 3000, 8, 3, 10, 0), (np.float32, 129, 128, 3, 3, 0), (np.float32, 700, 1, 2, 4, 1)])
def test_sharded_evaluate_on_one_device(dtype, N, N_max, s, p, cross):
    pos, q = inputs.uniform_cube(N, 302, dtype)
    P = fmm.Plan(dev(pos), p, N_max, s, 0.77, cross_level=cross)
    Po = O.Plan(pos, p, N_max, s, 0.77, cross_level=cross)
    uo, fo = Po.evaluate(q, fp32_rule=dtype == np.float32)
    tol = 1e-5 if dtype == np.float32 else 1e-11
    dq = dev(q)
    u_ref, f_ref = P.evaluate(dq)
    for n in (1, 2, 3, 8):
        u = torch.full_like(u_ref, float("nan"))
        f = torch.full_like(f_ref, float("nan"))
        for r in range(n):  # every shard's upward pass fills its leaf rows of the SAME plan: no exchange needed on one device
            fmm.fmm_evaluate_shard_upward(P.handle, n, r, dq)
        for r in range(n):
            fmm.fmm_evaluate_shard_downward(P.handle, n, r, u, f)
        torch.cuda.synchronize()
        un, fn = u.cpu().numpy(), f.cpu().numpy()
        assert np.all(np.isfinite(un)) and np.all(np.isfinite(fn)), n  # every particle written by exactly the shards together
        assert rel2(un, uo) <= tol and rel2(fn, fo) <= tol, (n, rel2(un, uo), rel2(fn, fo))
        assert rel2(un, u_ref.double().cpu().numpy()) <= 10 * (6e-8 if dtype == np.float32 else 1.2e-16) * 30
    # a shard writes its own particles only
    u = torch.full_like(u_ref, float("nan"))
    fmm.fmm_evaluate_shard_upward(P.handle, 2, 0, dq)
    fmm.fmm_evaluate_shard_upward(P.handle, 2, 1, dq)
    fmm.fmm_evaluate_shard_downward(P.handle, 2, 1, u, None)
    t = P.tree()
    lo, hi = fmm.fmm_shard_box_range(P.info["L"], s, 2, 1, P.info["L"])
    leaf0 = P.info["n_boxes"] - P.info["n_leaves"]
    own = np.zeros(N, bool)
    for leaf in range(lo, hi):
        st, c = t["box_start"][leaf0 + leaf], t["box_count"][leaf0 + leaf]
        own[t["perm"][st:st + c]] = True
    assert np.array_equal(np.isfinite(u.cpu().numpy()), own)
    P.close()


@pytest.mark.gpu
def test_two_plans_exchange_leaf_multipoles_like_two_ranks():
    """two plans of the same positions stand in for two ranks: each runs the upward pass of its shard, the leaf rows travel through
    fmm_plan_leaf_multipoles (what the all-gather of evaluate_sharded moves), each runs its downward pass"""
    pos, q = inputs.uniform_cube(30000, 303, np.float32)
    Po = O.Plan(pos, 8, 32, 3, 0.77)
    uo, fo = Po.evaluate(q, fp32_rule=True)
    plans = [fmm.Plan(dev(pos), 8, 32, 3, 0.77) for _ in range(2)]
    dq = dev(q)
    nl = plans[0].info["n_leaves"]
    kp = fmm.fmm_plan_leaf_multipoles(plans[0].handle, 0, 0, 0)
    assert kp == 84
    bounds = [fmm.fmm_shard_box_range(plans[0].info["L"], 3, 2, r, plans[0].info["L"]) for r in range(2)]
    rows = []
    for r in range(2):
        fmm.fmm_evaluate_shard_upward(plans[r].handle, 2, r, dq)
        buf = torch.empty((bounds[r][1] - bounds[r][0], kp), dtype=torch.float32, device="cuda")
        fmm.fmm_plan_leaf_multipoles(plans[r].handle, 0, bounds[r][0], bounds[r][1], buf)
        rows.append(buf)
    u = torch.full((30000,), float("nan"), dtype=torch.float32, device="cuda")
    f = torch.full((30000, 3), float("nan"), dtype=torch.float32, device="cuda")
    for r in range(2):
        o = 1 - r
        fmm.fmm_plan_leaf_multipoles(plans[r].handle, 1, bounds[o][0], bounds[o][1], rows[o])
        fmm.fmm_evaluate_shard_downward(plans[r].handle, 2, r, u, f)
    torch.cuda.synchronize()
    assert rel2(u.cpu().numpy(), uo) <= 1e-5 and rel2(f.cpu().numpy(), fo) <= 1e-5
    with pytest.raises(fmm.FmmError):
        fmm.fmm_evaluate_shard_upward(plans[0].handle, 2, 2, dq)
    for P in plans:
        P.close()
