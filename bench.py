#!/usr/bin/env python
"""bench.py -- FMM evaluate throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--sweep]

A "step" is one pass of the whole hot path (permute -> P2M -> M2M -> M2L -> L2L -> L2P -> P2P, SURVEY.md section 8(a) rows
a3-a10) over one charge vector on an existing plan (the paper times eval_potential on a cached hierarchy).
The default workload is BASELINE config 2 (N=1M uniform cube, fp32, p=8, s=3, N_max=128, theta=0.77); any name of
paper_2511_15269_b200/inputs.py works (configs 1-4, and the config-5 sweep points `cfg5_<cube|sphere>_<N>_<f32|f64>_p<p>_n<N_max>`).
Plan time is reported separately (`plan_ms`).  `value` times fmm_evaluate in its production (concurrent, forked-stream)
schedule; `stages` and `roofline.launch_ms` come from fmm_evaluate_profiled (same kernels back to back on one stream, CUDA
events between them), so the stage times add up to more than one step.  The L2 (126 MB) is flushed between timed steps by
writing a 512 MiB buffer; each step is timed with its own CUDA event pair on the launching stream, the flush lying outside.

N > 1 (torchrun): replicas only -- every rank evaluates its own independent problem of the same
shape; no data-path collective; value = particles of all ranks / max-over-ranks time; "scaling": "weak".

--impl reference: the CPU oracle (oracle/, test infrastructure) as it stands on the host cores (rank 0 only): ONE full evaluate
of the workload, timed (steps: 1 whatever --steps asks for: a second one would only repeat the first).
--sweep: the config-5 grid (N x p x dtype x point set x N_max) as a markdown table on stderr / --sweep-out and one JSON line.
"""
import argparse
import csv
import json
import os
import re
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FMM evaluate Mparticles/s at N=1M p=8 fp32"
UNIT = "Mparticles/s"
FP32_LANES_PER_SM, FP64_LANES_PER_SM, N_SM = 128, 64, 148
NCU_CSV = os.path.join(ROOT, "profiles", "r02_ncu_evaluate.csv")  # `ncu --page raw --csv` of one evaluate of the default workload
NCU_MD = os.path.join(ROOT, "profiles", "r02_ncu_evaluate.md")    # the command that made it, its workload and commit
TARGET_M2L_FRAC_HBM, TARGET_P2P_PIPE = 0.60, 0.50                   # BASELINE.json north_star


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


# ---------------------------------------------------------------- algorithmic work per unit
def m2l_nominal_fma_slots(p):
    """FMA-slot instructions of one rotation-based M2L as SURVEY.md section 8(d) counts them (three O(p^3) contractions of P(p)
    MACs, two azimuthal rotations per side, generation of the Wigner blocks).  NOMINAL: the kernels need fewer (the rotation blocks
    are constant matrices); what they execute is fmm_translation_work()."""
    P = (p + 1) * (2 * p * p + 4 * p + 3) / 3.0
    E = (p + 1) * (4 * p * p + 11 * p + 6) / 6.0
    return 3.0 * P + 4.0 * (p + 1) ** 2 + 2.5 * E


def m2l_bytes(p, esize, n_weak, n_targets):
    """algorithmic bytes of the M2L stage: per pair K*w source coefficients + 4 B list entry + 24 B source
    centre; per target box one read-modify-write of K*w."""
    K = (p + 1) ** 2
    return n_weak * (K * esize + 4 + 24) + n_targets * 2 * K * esize


P2P_FLOP_PER_PAIR = 20.0  # 3 sub, mul+2 FMA, rsqrt, 3 mul, 1+3 FMA, mask


def ncu_profile(workload):
    """Counters of the committed `ncu --set full` capture of one evaluate (profiles/r02_ncu_evaluate.csv, made by the command in
    profiles/r02_ncu_evaluate.md on the commit named there).  Returns {} when the capture is absent or belongs to another workload:
    nothing measured under a profiler is ever turned into a bench value, these only annotate the roofline line."""
    if not (os.path.exists(NCU_CSV) and os.path.exists(NCU_MD)):
        return {}
    md = open(NCU_MD).read()
    wl = re.search(r"workload:\s*`?([\w.]+)`?", md)
    commit = re.search(r"commit:\s*`?([0-9a-f]{7,40})`?", md)
    if not wl or wl.group(1) != workload:
        return {}
    rows = list(csv.reader(open(NCU_CSV)))
    hdr = rows[0]
    ix = {h: i for i, h in enumerate(hdr)}
    need = ["Kernel Name", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum"]
    if any(k not in ix for k in need):
        return {}
    unit = rows[1]

    def scale(col):
        u = unit[ix[col]].lower()
        return {"byte": 1.0, "kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9, "us": 1e-6, "ms": 1e-3, "ns": 1e-9, "s": 1.0, "usecond": 1e-6, "msecond": 1e-3,
                "nsecond": 1e-9, "second": 1.0}.get(u, 1.0)

    def f(r, col):
        try:
            return float(r[ix[col]].replace(",", "")) if col in ix else None
        except ValueError:
            return None

    out = {}
    for key, pat in (("m2l", r"xlate_\w+_k<\w+, (?:\(int\))?\d+, (?:\(int\))?1[,>]"), ("p2p", r"p2p_\w+_k<")):
        sel = [r for r in rows[2:] if len(r) == len(hdr) and re.search(pat, r[ix["Kernel Name"]])]
        if not sel:
            continue
        t = [f(r, "gpu__time_duration.sum") * scale("gpu__time_duration.sum") for r in sel]
        dram = sum((f(r, "dram__bytes_read.sum") + f(r, "dram__bytes_write.sum")) * scale("dram__bytes_read.sum") for r in sel)
        w = np.array(t) / sum(t)

        def wavg(col):
            v = [f(r, col) for r in sel]
            return float(np.dot(w, v)) if all(x is not None for x in v) else None

        fp = None
        cols = ["smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % o for o in ("ffma", "fmul", "fadd")]
        if all(c in ix for c in cols) and "sm__cycles_elapsed.max" in ix:
            fp = sum(sum(f(r, c) for c in cols) * f(r, "sm__cycles_elapsed.max") for r in sel)  # executed FP32 thread instructions
        out[key] = dict(launches=len(sel), time_s=sum(t), dram_bytes=dram, fp32_thread_inst=fp,
                        pipe_fma_pct=wavg("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active"),
                        pipe_fp64_pct=wavg("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"),
                        issue_active_pct=wavg("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                        stall_no_instruction=wavg("smsp__average_warps_issue_stalled_no_instruction_per_issue_active.ratio"))
    out["source"] = "profiles/r02_ncu_evaluate.csv (ncu --set full of one evaluate, commit %s; command in profiles/r02_ncu_evaluate.md)" % (
        commit.group(1) if commit else "unknown")
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, dev):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(dev), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [l.strip().split(", ") for l in open(self.f.name) if l.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def make_workload(name, rank):
    from paper_2511_15269_b200 import inputs
    c = dict(inputs.CONFIGS[name]) if name in inputs.CONFIGS else inputs.config5(name)
    c["seed"] = c["seed"] + 1000 * rank  # independent problem per replica
    inputs.CONFIGS["_bench"] = c
    pos, q, c = inputs.make("_bench")
    return pos, q, c


# ---------------------------------------------------------------- CPU oracle legs
def oracle_sampled(Po, q, c, n_leaves_sample, seed=0):
    """Bounded sample of the oracle as it stands: the full upward pass (P2M + M2M, which it always runs) plus M2L / L2L / L2P / P2P
    for n_leaves_sample random leaves and their ancestors (leaf mask), extrapolated to a full evaluate by the M2L pair count.
    Returns (estimated seconds per full evaluate, description)."""
    ls = Po.lists()
    rows = np.diff(ls["weak_off"])
    rng = np.random.default_rng(seed)
    mask = np.zeros(Po.n_leaves, np.uint8)
    mask[rng.choice(Po.n_leaves, min(n_leaves_sample, Po.n_leaves), replace=False)] = 1
    nch, L, s = 1 << c["s"], Po.L, c["s"]
    lvl_off = [sum(1 << (s * i) for i in range(l)) for l in range(L + 2)]
    boxes, pairs = np.flatnonzero(mask).astype(np.int64), 0
    for l in range(L, -1, -1):
        pairs += int(rows[lvl_off[l] + np.unique(boxes)].sum())
        boxes = boxes // nch
    t0 = time.perf_counter()
    Po.evaluate(q, leaf_mask=np.zeros_like(mask))
    t_up = time.perf_counter() - t0
    t0 = time.perf_counter()
    Po.evaluate(q, leaf_mask=mask)
    t_m = time.perf_counter() - t0
    pairs_total = int(rows.sum())
    t_full = t_up + max(t_m - t_up, 1e-9) * (pairs_total / max(pairs, 1))
    desc = ("full upward pass %.2f s + downward work for %d random leaves and their ancestors (%d of %d M2L pairs) %.2f s; "
            "t_full = t_up + t_down * pairs_total / pairs" % (t_up, int(mask.sum()), pairs, pairs_total, max(t_m - t_up, 0.0)))
    return t_full, desc


def oracle_baseline(pos, q, c, full=True, full_budget_s=420.0, one_thread=True):
    """cpu_baseline: the oracle (oracle/fmm_oracle.cpp, fp64, OpenMP) as it stands, on this box's host cores.  A full evaluate of
    the workload is MEASURED when the sampled estimate says it fits the budget; a 1-thread figure (comparable to the paper's
    single-core CPU column) is always a sampled estimate and labelled so."""
    from oracle import api as O
    N = pos.shape[0]
    t0 = time.perf_counter()
    Po = O.Plan(pos, c["p"], c["N_max"], c["s"], c["theta"])
    plan_s = time.perf_counter() - t0
    cores = O.num_threads()
    est, desc = oracle_sampled(Po, q, c, 16)
    out = dict(unit=UNIT, cores=cores, kind="oracle", plan_s=plan_s, sampled_estimate=dict(seconds_per_evaluate=est, value=N / est / 1e6, sample=desc))
    if full and est <= full_budget_s:
        t0 = time.perf_counter()
        u, _ = Po.evaluate(q)
        t_full = time.perf_counter() - t0
        assert bool(np.isfinite(u).all())
        out.update(value=N / t_full / 1e6, measured=True, seconds_per_evaluate=t_full,
                   sample="ONE full evaluate of all N = %d particles (potential + field), oracle/fmm_oracle.cpp as it stands, fp64, OpenMP %d threads: %.1f s "
                          "(the plan, %.1f s, is not in the time)" % (N, cores, t_full, plan_s))
    else:
        out.update(value=N / est / 1e6, measured=False, seconds_per_evaluate=est,
                   sample="SAMPLED ESTIMATE (%s; a full evaluate would take ~%.0f s): %s" % ("--cpu-sample" if not full else "over the %.0f s budget" % full_budget_s, est, desc))
    if one_thread:
        O.set_num_threads(1)
        try:
            est1, desc1 = oracle_sampled(Po, q, c, 2, seed=1)
        finally:
            O.set_num_threads(0)
        out["one_thread"] = dict(value=N / est1 / 1e6, unit=UNIT, cores=1, measured=False, seconds_per_evaluate=est1,
                                 sample="SAMPLED ESTIMATE on one thread: " + desc1)
    return out


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    pos, q, c = make_workload(args.workload, 0)
    N = pos.shape[0]
    b = oracle_baseline(pos, q, c, full=not args.cpu_sample, one_thread=False)
    t = b["seconds_per_evaluate"]
    line = dict(impl="reference", metric=METRIC, value=b["value"], unit=UNIT, n_gpus=args.gpus, steps=1, steps_requested=args.steps, warmup=0,
                warmup_requested=args.warmup, ms_per_step=t * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=args.workload, N=N, p=c["p"], s=c["s"], N_max=c["N_max"], theta=c["theta"]),
                cpu_baseline=dict(value=b["value"], unit=UNIT, cores=b["cores"], kind="oracle", measured=b["measured"], sample=b["sample"],
                                  sampled_estimate=b["sampled_estimate"], plan_s=b["plan_s"]),
                e2e=dict(value=b["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


def aggregate_over_ranks(total_ms, e2e_ms, N, steps, world, device):
    """Replicas: every rank evaluates its own problem of N particles; the job's time is the MAX over ranks
    of the device time of `steps` steps (and of one end-to-end step), the job's value the particles of ALL ranks over that time.
    Returns (ms_per_step, Mparticles/s, e2e ms per step, e2e Mparticles/s).  Needs an initialised process group if world > 1."""
    import torch
    import torch.distributed as dist
    tmax = torch.tensor([total_ms, e2e_ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    total_ms_max, e2e_ms_max = float(tmax[0]), float(tmax[1])
    ms_per_step = total_ms_max / steps
    return ms_per_step, world * N / ms_per_step / 1e3, e2e_ms_max, world * N / e2e_ms_max / 1e3


def time_evaluates(fmm, handle, d_q, d_u, d_f, flush, n, warm=3):
    """mean ms of n evaluates, each in its own CUDA-event pair, L2 flushed in between (outside the pairs)"""
    import torch
    for _ in range(warm):
        flush.zero_()
        fmm.fmm_evaluate(handle, d_q, d_u, d_f)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    for a, b in ev:
        flush.zero_()
        a.record()
        fmm.fmm_evaluate(handle, d_q, d_u, d_f)
        b.record()
    torch.cuda.synchronize()
    return np.array([a.elapsed_time(b) for a, b in ev])


# ---------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2511_15269_b200 import fmm

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    fmm.lib()  # fail loudly if the CUDA extension is missing
    peaks = load_peaks()

    # --sharded (N > 1): ONE problem, its targets sharded over the ranks (fmm.evaluate_sharded: upward pass of the own leaves, one NCCL
    # all-gather of the leaf multipoles, downward pass of the own targets): "scaling": "strong".  Default: independent replicas.
    sharded = bool(args.sharded) and world > 1
    pos, q, c = make_workload(args.workload, 0 if sharded else rank)
    N = pos.shape[0]
    tdt = torch.float32 if pos.dtype == np.float32 else torch.float64
    esize = pos.dtype.itemsize
    d_pos = torch.from_numpy(pos).cuda()
    d_q = torch.from_numpy(q).cuda()
    P = fmm.Plan(d_pos, c["p"], c["N_max"], c["s"], c["theta"], cross_level=args.cross_level)
    plan_ms = P.timings()
    info = P.info
    d_u = torch.empty(N, dtype=tdt, device="cuda")
    d_f = torch.empty((N, 3), dtype=tdt, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    launches = fmm.fmm_plan_launches(P.handle)

    def step():
        if sharded:
            fmm.evaluate_sharded(P.handle, info["n_leaves"], d_q, d_u, d_f)
        else:
            fmm.fmm_evaluate(P.handle, d_q, d_u, d_f)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()
        a.record()
        step()
        b.record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = float(step_ms.sum())

    # instrumented pass over the same steps: CUDA events between the stages (fmm_evaluate_profiled), L2 flushed as above
    n_prof = min(args.steps, 50)
    stage = {}
    for _ in range(n_prof):
        flush.zero_()
        ms = fmm.fmm_evaluate_profiled(P.handle, d_q, d_u, d_f)
        for k, v in ms.items():
            stage.setdefault(k, []).append(v)
    stage_ms = {k: float(np.mean(v)) for k, v in stage.items()}
    clocks = sampler.stop() if sampler else None

    # end to end through the C-ABI with HOST buffers (pinned): H2D of the charges and D2H of potential+field inside the timed region
    h_q = torch.from_numpy(q).pin_memory()
    h_u = torch.empty(N, dtype=tdt).pin_memory()
    h_f = torch.empty((N, 3), dtype=tdt).pin_memory()
    n_e2e = min(args.steps, 30)
    for _ in range(3):
        fmm.fmm_evaluate_host(P.handle, h_q, h_u, h_f)
    barrier()
    e2e_s = 0.0
    for _ in range(n_e2e):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        fmm.fmm_evaluate_host(P.handle, h_q, h_u, h_f)  # synchronises before returning
        e2e_s += time.perf_counter() - t0
    e2e_sync_ms = e2e_s * 1e3 / n_e2e
    assert bool(torch.isfinite(h_u).all()) and bool(torch.isfinite(h_f).all())
    # the same path as a two-deep pipeline (fmm_evaluate_host_submit / _wait): every step still copies its charges in and its
    # potential + field out, but the copies of one step cross PCIe beside the kernels of the next.  Throughput over n_e2e steps,
    # wall clock, nothing in flight before or after.  No flush inside the loop: one step streams more than the L2 holds.
    h_u2 = torch.empty(N, dtype=tdt).pin_memory()
    h_f2 = torch.empty((N, 3), dtype=tdt).pin_memory()
    outs = [(h_u, h_f), (h_u2, h_f2)]

    def pipelined(n):
        for k in range(n):
            if k >= 2:
                fmm.fmm_evaluate_host_wait(P.handle)
            fmm.fmm_evaluate_host_submit(P.handle, h_q, *outs[k & 1])
        for _ in range(min(n, 2)):
            fmm.fmm_evaluate_host_wait(P.handle)

    pipelined(4)
    ref_u, ref_f = h_u.clone(), h_f.clone()
    barrier()
    flush.zero_()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    pipelined(n_e2e)
    e2e_ms = (time.perf_counter() - t0) * 1e3 / n_e2e
    for a in (h_u, h_f, h_u2, h_f2):
        assert bool(torch.isfinite(a).all())
    assert float((h_u2 - ref_u).abs().max()) <= 1e-4 * float(ref_u.abs().max()) and float((h_f2 - ref_f).abs().max()) <= 1e-4 * float(ref_f.abs().max())

    extras = rank == 0 and not args.no_extras
    n_x = min(args.steps, 50)
    # the same workload with the paper's level-marching lists (fmm_admissibility.cross_level = 1): fewer M2L
    # pairs at the same theta, somewhat larger error.  Reported beside the headline, not instead of it.
    alt = None
    if extras:
        Pa = fmm.Plan(d_pos, c["p"], c["N_max"], c["s"], c["theta"], cross_level=1 - args.cross_level)
        ms_alt = float(time_evaluates(fmm, Pa.handle, d_q, d_u, d_f, flush, n_x).mean())
        alt = dict(cross_level=1 - args.cross_level, n_weak=Pa.info["n_weak"], n_strong=Pa.info["n_strong"], ms_per_step=ms_alt,
                   value=N / ms_alt / 1e3, unit=UNIT, steps=n_x, plan_ms=Pa.timings())
        Pa.close()

    # potential only (what the paper's eval_potential returns and its Table III times): d_field = NULL skips the field
    # arithmetic of P2P and L2P.  Reported beside the headline (which is potential + field, as north_star asks).
    pot_only = None
    if extras:
        ms_po = float(time_evaluates(fmm, P.handle, d_q, d_u, None, flush, n_x).mean())
        pot_only = dict(ms_per_step=ms_po, value=N / ms_po / 1e3, unit=UNIT, steps=n_x)

    # re-planning cost for changed positions (the paper pays minutes of JIT whenever positions change): wall time of
    # plan create + destroy on the same positions with a warm memory pool, synchronised on both sides
    replan = None
    if extras:
        ts = []
        for _ in range(6):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            Pr = fmm.Plan(d_pos, c["p"], c["N_max"], c["s"], c["theta"], cross_level=args.cross_level)
            torch.cuda.synchronize()
            ts.append((time.perf_counter() - t0) * 1e3)
            last = Pr.timings()
            Pr.close()
        replan = dict(wall_ms_mean=float(np.mean(ts[1:])), wall_ms_min=float(np.min(ts[1:])), device_ms=last, n=5)

    # the paper's second workload: the same sources evaluated at N separate targets (uniform in the unit cube, seed 102)
    st_line = None
    if extras:
        tgt = np.ascontiguousarray(np.random.default_rng(102).random((N, 3)).astype(pos.dtype))
        d_tgt = torch.from_numpy(tgt).cuda()
        Pt = fmm.PlanTargets(d_pos, d_tgt, c["p"], c["N_max"], c["s"], c["theta"])
        d_ut = torch.empty(N, dtype=tdt, device="cuda")
        d_ft = torch.empty((N, 3), dtype=tdt, device="cuda")
        ms_st = float(time_evaluates(fmm, Pt.handle, d_q, d_ut, d_ft, flush, n_x).mean())
        st_line = dict(n_sources=N, n_targets=N, n_weak=Pt.info["n_weak"], n_strong=Pt.info["n_strong"], n_p2p_pairs=Pt.info["n_p2p_pairs"],
                       ms_per_step=ms_st, value=N / ms_st / 1e3, unit="M targets/s", steps=n_x, plan_ms=Pt.timings())
        Pt.close()
        del d_tgt, d_ut, d_ft

    ms_per_step, value, e2e_ms_max, e2e_value = aggregate_over_ranks(total_ms, e2e_ms, N, args.steps, world, "cuda")
    if sharded:  # one problem of N particles, not `world` of them
        value, e2e_value = value / world, e2e_value / world
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel; both far-field and near-field leaders are reported under "stages"
    sm_hz = peaks["sm_max_mhz"] * 1e6
    lanes = FP32_LANES_PER_SM if esize == 4 else FP64_LANES_PER_SM
    alu_peak_tflops = N_SM * lanes * 2 * sm_hz / 1e12
    fma, mul, add = fmm.fmm_translation_work(c["p"], P.dtype, 1)            # what one M2L executes in the kernels that ran
    m2l_flop_exec = (2.0 * fma + mul + add) * info["n_weak"]
    m2l_inst_exec = float(fma + mul + add)
    m2l_flop_nominal = 2.0 * m2l_nominal_fma_slots(c["p"]) * info["n_weak"]
    m2l_b = m2l_bytes(c["p"], esize, info["n_weak"], info["n_boxes"])
    p2p_flops = P2P_FLOP_PER_PAIR * info["n_p2p_pairs"]
    t_m2l, t_p2p = stage_ms["m2l"] * 1e-3, stage_ms["p2p"] * 1e-3
    ncu = ncu_profile(args.workload) if args.cross_level == 0 else {}
    stages = dict(stage_ms)
    stages.update(m2l_tflops_executed=m2l_flop_exec / t_m2l / 1e12 if t_m2l > 0 and m2l_inst_exec > 0 else None,
                  m2l_tflops_nominal_survey=m2l_flop_nominal / t_m2l / 1e12 if t_m2l > 0 else None,
                  m2l_fp_inst_per_pair=m2l_inst_exec, m2l_fp_inst_per_pair_nominal_survey=m2l_nominal_fma_slots(c["p"]),
                  m2l_hbm_equiv_gbs=m2l_b / t_m2l / 1e9 if t_m2l > 0 else None,
                  p2p_tflops=p2p_flops / t_p2p / 1e12, p2p_gpairs_per_s=info["n_p2p_pairs"] / t_p2p / 1e9)
    stages["m2l_frac_hbm"] = stages["m2l_hbm_equiv_gbs"] / peaks["hbm_gbs"] if stages["m2l_hbm_equiv_gbs"] else None
    stages["m2l_frac_alu_executed"] = stages["m2l_tflops_executed"] / alu_peak_tflops if stages["m2l_tflops_executed"] else None
    stages["m2l_frac_alu_nominal_survey"] = stages["m2l_tflops_nominal_survey"] / alu_peak_tflops if stages["m2l_tflops_nominal_survey"] else None
    stages["p2p_frac_alu"] = stages["p2p_tflops"] / alu_peak_tflops
    stages["m2l_pipe_active_ncu"] = (ncu.get("m2l", {}).get("pipe_fma_pct" if esize == 4 else "pipe_fp64_pct") or 0) / 100.0 or None
    stages["p2p_pipe_active_ncu"] = (ncu.get("p2p", {}).get("pipe_fma_pct" if esize == 4 else "pipe_fp64_pct") or 0) / 100.0 or None
    targets = dict(m2l_frac_hbm=dict(target=TARGET_M2L_FRAC_HBM, value=stages["m2l_frac_hbm"],
                                     target_met=bool(stages["m2l_frac_hbm"] and stages["m2l_frac_hbm"] >= TARGET_M2L_FRAC_HBM),
                                     note="algorithmic bytes / time over the measured HBM copy bandwidth (an equivalent: the coefficient arrays are L2-resident)"),
                   p2p_pipe=dict(target=TARGET_P2P_PIPE, value_flop_count=stages["p2p_frac_alu"], value_ncu_pipe=stages["p2p_pipe_active_ncu"],
                                 target_met_flop_count=bool(stages["p2p_frac_alu"] >= TARGET_P2P_PIPE),
                                 target_met_ncu_pipe=(None if stages["p2p_pipe_active_ncu"] is None else bool(stages["p2p_pipe_active_ncu"] >= TARGET_P2P_PIPE)),
                                 note="north_star names the ncu pipe-utilisation counter as the evidence; the flop-count fraction uses 20 flop per pair"))
    dom = "m2l" if stage_ms["m2l"] >= stage_ms["p2p"] else "p2p"
    achieved = stages["m2l_tflops_executed"] if dom == "m2l" else stages["p2p_tflops"]
    nprof = ncu.get(dom, {})
    per_pair_ncu = None
    if dom == "m2l" and nprof.get("fp32_thread_inst"):
        per_pair_ncu = nprof["fp32_thread_inst"] / info["n_weak"]
    roofline = dict(kernel=dom, bound="alu", achieved=achieved, peak=alu_peak_tflops, unit="TFLOP/s", frac=(achieved / alu_peak_tflops) if achieved else None,
                    achieved_kind=("executed flop: (2 fma + mul + add) of fmm_translation_work(p) x n_weak / launch time" if dom == "m2l"
                                   else "20 flop per particle pair x n_p2p_pairs / launch time"),
                    traffic=nprof.get("dram_bytes"), traffic_source=ncu.get("source") if nprof else None,
                    pipe_active=(nprof.get("pipe_fma_pct" if esize == 4 else "pipe_fp64_pct") or 0) / 100.0 or None,
                    issue_active=(nprof.get("issue_active_pct") or 0) / 100.0 or None, stall_no_instruction=nprof.get("stall_no_instruction"),
                    executed_fp32_per_pair=m2l_inst_exec if dom == "m2l" else None, executed_fp32_per_pair_ncu=per_pair_ncu,
                    nominal_algorithmic_tflops=stages["m2l_tflops_nominal_survey"] if dom == "m2l" else None,
                    nominal_frac=stages["m2l_frac_alu_nominal_survey"] if dom == "m2l" else None,
                    algorithmic_bytes=m2l_b if dom == "m2l" else None,
                    peak_source="148 SM x %d lanes x 2 x %.0f MHz (DESIGN.md; an FFMA micro-benchmark reached 98%% of the FP32 figure)" % (lanes, peaks["sm_max_mhz"]),
                    launch_ms=stage_ms[dom], launches_per_step=1,
                    launch_ms_source="CUDA events around the kernel in fmm_evaluate_profiled (serial schedule, one launch), mean of %d steps" % n_prof,
                    hbm_peak_gbs=peaks["hbm_gbs"], hbm_peak_source=peaks["source"])

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        cpu_baseline = oracle_baseline(pos, q, c, full=not args.cpu_sample)

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3), ms_per_step=ms_per_step,
                higher_is_better=True, scaling="strong" if sharded else "weak", vs_baseline=None, dtype="f32" if esize == 4 else "f64", data="synthetic",
                config=dict(workload=args.workload, N=N, p=c["p"], s=c["s"], N_max=c["N_max"], theta=c["theta"], cross_level=args.cross_level,
                            outputs="potential+field",
                            L=info["L"], n_boxes=info["n_boxes"], n_weak=info["n_weak"], n_strong=info["n_strong"], n_p2p_pairs=info["n_p2p_pairs"],
                            l2="flushed between timed steps (512 MiB memset outside the event pairs)", parallelism=("targets sharded x%d (one all-gather of leaf multipoles per step; e2e is the unsharded host path of each rank)" % world) if sharded
                            else "replicas x%d" % world,
                            schedule="concurrent: P2P, the tree passes (M2M, upper-level M2L, L2L) and the leaf-level M2L on three forked streams"),
                clocks=clocks, e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=N * esize, d2h_bytes_per_step=N * 4 * esize,
                                        ms_per_step=e2e_ms_max, steps=n_e2e, api="fmm_evaluate_host_submit / fmm_evaluate_host_wait, two calls in flight, pinned host buffers",
                                        latency_ms_single_call=e2e_sync_ms, latency_api="fmm_evaluate_host (synchronous, L2 flushed before each call)"),
                gpu_launches=launches * args.steps, gpu_launches_per_step=launches, roofline=roofline, stages=stages, targets=targets, plan_ms=plan_ms,
                alt_lists=alt, potential_only=pot_only, separate_targets=st_line, replan=replan, min_ms_per_step=float(step_ms.min()),
                wall_ms_per_step_incl_flush=t_wall * 1e3 / args.steps, cpu_baseline=cpu_baseline)
    print(json.dumps(line), flush=True)
    P.close()
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------- config-5 sweep (one GPU)
def run_sweep(args):
    """BASELINE config 5 (the paper's Figs. 5-10 shape): N x p x dtype x point set x N_max.  For every point one
    plan (timed), 3 warm-up evaluates, then `--steps` evaluates in CUDA-event pairs (L2 flushed between them); minimum and mean are
    reported as the paper does, plus the serial per-stage times."""
    import itertools
    import torch
    from paper_2511_15269_b200 import fmm
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep: no CUDA device")
    sets = args.sweep_sets.split(",")
    Ns = [int(float(x)) for x in args.sweep_N.split(",")]
    ps = [int(x) for x in args.sweep_p.split(",")]
    dts = args.sweep_dtype.split(",")
    nmaxs = [int(x) for x in args.sweep_nmax.split(",")]
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    lines = ["| workload | L | weak pairs | P2P pairs | plan ms | evaluate min ms | mean ms | Mparticles/s (min) | M2L ms | P2P ms | other ms |",
             "|---|---|---|---|---|---|---|---|---|---|---|"]
    points = []
    for kind, N, dt, p, nmax in itertools.product(sets, Ns, dts, ps, nmaxs):
        name = "cfg5_%s_%d_%s_p%d_n%d" % (kind, N, dt, p, nmax)
        try:
            pos, q, c = make_workload(name, 0)
            tdt = torch.float32 if dt == "f32" else torch.float64
            d_pos, d_q = torch.from_numpy(pos).cuda(), torch.from_numpy(q).cuda()
            P = fmm.Plan(d_pos, c["p"], c["N_max"], c["s"], c["theta"])
            d_u = torch.empty(N, dtype=tdt, device="cuda")
            d_f = torch.empty((N, 3), dtype=tdt, device="cuda")
            ts = time_evaluates(fmm, P.handle, d_q, d_u, d_f, flush, args.steps)
            flush.zero_()
            st = fmm.fmm_evaluate_profiled(P.handle, d_q, d_u, d_f)
            ok = bool(torch.isfinite(d_u).all()) and bool(torch.isfinite(d_f).all())
            r = dict(workload=name, L=P.info["L"], n_weak=P.info["n_weak"], n_p2p_pairs=P.info["n_p2p_pairs"], plan_ms=P.timings()["total"],
                     min_ms=float(ts.min()), mean_ms=float(ts.mean()), value=N / float(ts.min()) / 1e3, m2l_ms=st["m2l"], p2p_ms=st["p2p"],
                     other_ms=st["total"] - st["m2l"] - st["p2p"], finite=ok)
            P.close()
            del d_pos, d_q, d_u, d_f
        except Exception as e:  # report and go on: one failing point must not hide the others
            r = dict(workload=name, failed=str(e)[:120])
        points.append(r)
        if "failed" in r:
            lines.append("| %s | failed: %s |" % (name, r["failed"]))
        else:
            lines.append("| %s | %d | %.3g | %.3g | %.1f | %.3f | %.3f | %.1f | %.3f | %.3f | %.3f |%s" % (
                name, r["L"], r["n_weak"], r["n_p2p_pairs"], r["plan_ms"], r["min_ms"], r["mean_ms"], r["value"], r["m2l_ms"], r["p2p_ms"], r["other_ms"],
                "" if r["finite"] else " non-finite output"))
        print(lines[-1], file=sys.stderr, flush=True)
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            f.write("\n".join(lines) + "\n")
    print(json.dumps(dict(metric="config-5 sweep: FMM evaluate Mparticles/s (min of %d)" % args.steps, unit=UNIT, n_gpus=1, steps=args.steps, data="synthetic",
                          points=points)), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2_cube1M_f32")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample", action="store_true", help="cpu_baseline / --impl reference: the bounded sample only, no full oracle evaluate")
    ap.add_argument("--cross-level", type=int, default=0, choices=[0, 1],
                    help="interaction lists of the timed plan: 0 = same-level (paper default, PAPER.md:72-74), 1 = level marching (PAPER.md:82-89)")
    ap.add_argument("--no-extras", "--no-alt-lists", dest="no_extras", action="store_true",
                    help="skip the extra measurements (the other list kind, potential only, re-plan, separate targets)")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: one problem with its targets sharded over the ranks (strong scaling) instead of independent replicas")
    ap.add_argument("--sweep", action="store_true", help="run the config-5 grid instead of the headline")
    ap.add_argument("--sweep-out", default=None, help="write the markdown table of --sweep here")
    ap.add_argument("--sweep-sets", default="cube,sphere")
    ap.add_argument("--sweep-N", default="1e4,1e5,1e6,1e7")
    ap.add_argument("--sweep-p", default="4,8,12")
    ap.add_argument("--sweep-dtype", default="f32,f64")
    ap.add_argument("--sweep-nmax", default="32,128,512")
    args = ap.parse_args()
    if args.sweep:
        if args.steps == 100:
            args.steps = 10
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
