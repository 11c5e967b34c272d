#!/usr/bin/env python
"""bench.py -- FMM evaluate throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path (permute -> P2M -> M2M -> M2L -> L2L -> L2P -> P2P, SURVEY.md section 8(a) rows
a3-a10) over one charge vector on an existing plan (the paper times eval_potential on a cached hierarchy).
The workload is BASELINE config 2 (N=1M uniform cube, fp32, p=8, s=3, N_max=128, theta=0.77); plan time is reported
separately in the JSON (`plan_ms`).  `value` times fmm_evaluate in its production (concurrent, forked-stream) schedule;
`stages` and `roofline.launch_ms` come from fmm_evaluate_profiled (same kernels back to back on one stream, CUDA events
between them), so the stage times add up to more than one step.  The L2 (126 MB) is flushed between timed steps by writing a 512 MiB buffer; each step
is timed with its own CUDA event pair on the launching stream, the flush lying outside the pairs.

N > 1 (torchrun): replicas only -- every rank evaluates its own independent problem of the same
shape; no data-path collective; value = particles of all ranks / max-over-ranks time; "scaling": "weak".

--impl reference: the CPU oracle (oracle/, test infrastructure) timed as it stands on the host cores (rank 0 only).
"""
import argparse
import json
import os
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
FP32_LANES_PER_SM, N_SM = 128, 148


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


# ---------------------------------------------------------------- algorithmic work per unit
def m2l_fma_slots(p):
    """FMA-slot instructions of one rotation-based M2L: three O(p^3) contractions (two polar
    rotations + z-shift) of P(p) MACs each, two azimuthal rotations on each side, generation of the rotation blocks."""
    P = (p + 1) * (2 * p * p + 4 * p + 3) / 3.0
    E = (p + 1) * (4 * p * p + 11 * p + 6) / 6.0
    return 3.0 * P + 4.0 * (p + 1) ** 2 + 2.5 * E


def m2l_bytes(p, esize, n_weak, n_targets):
    """algorithmic bytes of the M2L stage: per pair K*w source coefficients + 4 B list entry + 24 B source centre;
    per target box with a non-empty row one read-modify-write of K*w."""
    K = (p + 1) ** 2
    return n_weak * (K * esize + 4 + 24) + n_targets * 2 * K * esize


P2P_FLOP_PER_PAIR = 20.0  # 3 sub, mul+2 FMA, rsqrt, 3 mul, 1+3 FMA, mask

# dram__bytes_read.sum + dram__bytes_write.sum per evaluate of the named kernel, from the committed `ncu --set full` capture
# profiles/r01_ncu_full_evaluate.md (M2L = leaf-level launch 71.27 MB + upper-levels launch 8.66 MB)
NCU_DRAM_BYTES = {"cfg2_cube1M_f32": {"m2l": 79.58e6, "p2p": 37.13e6}}


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
    c = dict(inputs.CONFIGS[name])
    c["seed"] = c["seed"] + 1000 * rank  # independent problem per replica
    inputs.CONFIGS["_bench"] = c
    pos, q, c = inputs.make("_bench")
    return pos, q, c


# ---------------------------------------------------------------- CPU oracle legs
def oracle_sample(pos, q, c, n_leaves_sample, seed=0):
    """Times the oracle as it stands on a bounded sample: one evaluate restricted (leaf mask) to n_leaves_sample random
    leaves.  The oracle always runs its full upward pass (P2M + M2M); the downward work is proportional to the M2L pairs of
    the needed boxes.  Returns (seconds_up, seconds_masked, pairs_done, pairs_total, particles_done, threads)."""
    from oracle import api as O
    Po = O.Plan(pos, c["p"], c["N_max"], c["s"], c["theta"])
    ls = Po.lists()
    rows = np.diff(ls["weak_off"])
    rng = np.random.default_rng(seed)
    mask = np.zeros(Po.n_leaves, np.uint8)
    mask[rng.choice(Po.n_leaves, min(n_leaves_sample, Po.n_leaves), replace=False)] = 1
    nch, L, s = 1 << c["s"], Po.L, c["s"]
    need = np.flatnonzero(mask).astype(np.int64)
    pairs, lvl_off = 0, [sum(1 << (s * i) for i in range(l)) for l in range(L + 2)]
    boxes = need.copy()
    for l in range(L, -1, -1):
        pairs += int(rows[lvl_off[l] + np.unique(boxes)].sum())
        boxes = boxes // nch
    t = Po.tree()
    done = int(t["box_count"][lvl_off[L] + need].sum())
    return Po, mask, pairs, int(rows.sum()), done


def time_oracle_step(Po, q, mask):
    t0 = time.perf_counter()
    Po.evaluate(q, leaf_mask=np.zeros_like(mask))
    t_up = time.perf_counter() - t0
    t0 = time.perf_counter()
    Po.evaluate(q, leaf_mask=mask)
    t_m = time.perf_counter() - t0
    return t_up, t_m


def extrapolate(N, t_up, t_m, pairs, pairs_total):
    t_full = t_up + max(t_m - t_up, 1e-9) * (pairs_total / max(pairs, 1))
    return N / t_full / 1e6, t_full


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import api as O
    pos, q, c = make_workload(args.workload, 0)
    N = pos.shape[0]
    Po, mask, pairs, pairs_total, done = oracle_sample(pos, q, c, args.ref_leaves)
    t_up, t_m = time_oracle_step(Po, q, mask)  # first warm-up, also sizes the run
    budget, t_step = 150.0, t_up + t_m
    warm = max(0, min(args.warmup - 1, int(20.0 / t_step)))
    steps = max(1, min(args.steps, int(budget / t_step)))
    for _ in range(warm):
        time_oracle_step(Po, q, mask)
    tu, tm = [], []
    for _ in range(steps):
        a, b = time_oracle_step(Po, q, mask)
        tu.append(a)
        tm.append(b)
    val, t_full = extrapolate(N, float(np.mean(tu)), float(np.mean(tm)), pairs, pairs_total)
    cores = O.num_threads()
    sample = ("oracle/fmm_oracle.cpp as it stands, fp64, OpenMP %d threads: per step one full upward pass (P2M+M2M, %.2f s) + M2L/L2L/L2P/P2P "
              "for %d random leaves and their ancestors (%d of %d M2L pairs, %d particles, %.2f s); value = N / (t_up + t_down * pairs_total/pairs)"
              % (cores, np.mean(tu), int(mask.sum()), pairs, pairs_total, done, np.mean(tm) - np.mean(tu)))
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=steps, steps_requested=args.steps, warmup=warm + 1,
                ms_per_step=t_full * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=args.workload, N=N, p=c["p"], s=c["s"], N_max=c["N_max"], theta=c["theta"]),
                cpu_baseline=dict(value=val, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
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

    pos, q, c = make_workload(args.workload, rank)
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

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        fmm.fmm_evaluate(P.handle, d_q, d_u, d_f)
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()
        a.record()
        fmm.fmm_evaluate(P.handle, d_q, d_u, d_f)
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
    e2e_ms = e2e_s * 1e3 / n_e2e
    assert bool(torch.isfinite(h_u).all()) and bool(torch.isfinite(h_f).all())

    # the same workload with the paper's level-marching lists (fmm_admissibility.cross_level = 1): fewer M2L
    # pairs at the same theta, somewhat larger error.  Reported beside the headline, not instead of it.
    alt = None
    if rank == 0 and not args.no_alt_lists:
        Pa = fmm.Plan(d_pos, c["p"], c["N_max"], c["s"], c["theta"], cross_level=1 - args.cross_level)
        n_alt = min(args.steps, 50)
        for _ in range(3):
            flush.zero_()
            fmm.fmm_evaluate(Pa.handle, d_q, d_u, d_f)
        eva = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_alt)]
        for a, b in eva:
            flush.zero_()
            a.record()
            fmm.fmm_evaluate(Pa.handle, d_q, d_u, d_f)
            b.record()
        torch.cuda.synchronize()
        ms_alt = float(np.mean([a.elapsed_time(b) for a, b in eva]))
        alt = dict(cross_level=1 - args.cross_level, n_weak=Pa.info["n_weak"], n_strong=Pa.info["n_strong"], ms_per_step=ms_alt,
                   value=N / ms_alt / 1e3, unit=UNIT, steps=n_alt, plan_ms=Pa.timings())
        Pa.close()

    # potential only (what the paper's eval_potential returns and its Table III times): d_field = NULL skips the field
    # arithmetic of P2P and L2P.  Reported beside the headline (which is potential + field, as north_star asks).
    pot_only = None
    if rank == 0 and not args.no_alt_lists:
        n_po = min(args.steps, 50)
        for _ in range(3):
            flush.zero_()
            fmm.fmm_evaluate(P.handle, d_q, d_u, None)
        evp = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_po)]
        for a, b in evp:
            flush.zero_()
            a.record()
            fmm.fmm_evaluate(P.handle, d_q, d_u, None)
            b.record()
        torch.cuda.synchronize()
        ms_po = float(np.mean([a.elapsed_time(b) for a, b in evp]))
        pot_only = dict(ms_per_step=ms_po, value=N / ms_po / 1e3, unit=UNIT, steps=n_po)

    # re-planning cost for changed positions (the paper pays minutes of JIT whenever positions change): wall time of
    # plan create + destroy on the same positions with a warm memory pool, synchronised on both sides
    replan = None
    if rank == 0 and not args.no_alt_lists:
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
    if rank == 0 and not args.no_alt_lists:
        tgt = np.ascontiguousarray(np.random.default_rng(102).random((N, 3)).astype(pos.dtype))
        d_tgt = torch.from_numpy(tgt).cuda()
        Pt = fmm.PlanTargets(d_pos, d_tgt, c["p"], c["N_max"], c["s"], c["theta"])
        d_ut = torch.empty(N, dtype=tdt, device="cuda")
        d_ft = torch.empty((N, 3), dtype=tdt, device="cuda")
        n_st = min(args.steps, 50)
        for _ in range(3):
            flush.zero_()
            fmm.fmm_evaluate(Pt.handle, d_q, d_ut, d_ft)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_st)]
        for a, b in evs:
            flush.zero_()
            a.record()
            fmm.fmm_evaluate(Pt.handle, d_q, d_ut, d_ft)
            b.record()
        torch.cuda.synchronize()
        ms_st = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        st_line = dict(n_sources=N, n_targets=N, n_weak=Pt.info["n_weak"], n_strong=Pt.info["n_strong"], n_p2p_pairs=Pt.info["n_p2p_pairs"],
                       ms_per_step=ms_st, value=N / ms_st / 1e3, unit="M targets/s", steps=n_st, plan_ms=Pt.timings())
        Pt.close()
        del d_tgt, d_ut, d_ft

    ms_per_step, value, e2e_ms_max, e2e_value = aggregate_over_ranks(total_ms, e2e_ms, N, args.steps, world, "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (both far-field and near-field leaders are reported under "stages")
    sm_hz = peaks["sm_max_mhz"] * 1e6
    fp32_peak_tflops = N_SM * FP32_LANES_PER_SM * 2 * sm_hz / 1e12
    n_tgt_rows = info["n_boxes"]
    m2l_flops = 2.0 * m2l_fma_slots(c["p"]) * info["n_weak"]
    m2l_b = m2l_bytes(c["p"], esize, info["n_weak"], n_tgt_rows)
    p2p_flops = P2P_FLOP_PER_PAIR * info["n_p2p_pairs"]
    stages = dict(stage_ms)
    stages.update(m2l_tflops=m2l_flops / (stage_ms["m2l"] * 1e-3) / 1e12 if stage_ms["m2l"] > 0 else 0.0,
                  m2l_hbm_equiv_gbs=m2l_b / (stage_ms["m2l"] * 1e-3) / 1e9 if stage_ms["m2l"] > 0 else 0.0,
                  p2p_tflops=p2p_flops / (stage_ms["p2p"] * 1e-3) / 1e12,
                  p2p_gpairs_per_s=info["n_p2p_pairs"] / (stage_ms["p2p"] * 1e-3) / 1e9)
    stages["m2l_frac_hbm"] = stages["m2l_hbm_equiv_gbs"] / peaks["hbm_gbs"]
    stages["m2l_frac_fp32"] = stages["m2l_tflops"] / fp32_peak_tflops
    stages["p2p_frac_fp32"] = stages["p2p_tflops"] / fp32_peak_tflops
    dom = "m2l" if stage_ms["m2l"] >= stage_ms["p2p"] else "p2p"
    roofline = dict(kernel=dom, bound="alu", achieved=stages[dom + "_tflops"], peak=fp32_peak_tflops, unit="TFLOP/s",
                    frac=stages[dom + "_tflops"] / fp32_peak_tflops, traffic=NCU_DRAM_BYTES.get(args.workload, {}).get(dom),
                    traffic_source="profiles/r01_ncu_full_evaluate.md (ncu --set full, dram bytes read+write of this kernel per evaluate)",
                    algorithmic_bytes=m2l_b if dom == "m2l" else None,
                    peak_source="148 SM x 128 FP32 lanes x 2 x %.0f MHz (DESIGN.md; FFMA micro-benchmark reached 98%% of it)" % peaks["sm_max_mhz"],
                    launch_ms=stage_ms[dom], launches_per_step=1,
                    launch_ms_source="CUDA events around the kernel in fmm_evaluate_profiled (serial schedule, one launch), mean of %d steps" % n_prof,
                    hbm_peak_gbs=peaks["hbm_gbs"], hbm_peak_source=peaks["source"])

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import api as O
        Po, mask, pairs, pairs_total, done = oracle_sample(pos, q, c, args.cpu_leaves)
        t_up, t_m = time_oracle_step(Po, q, mask)
        val, t_full = extrapolate(N, t_up, t_m, pairs, pairs_total)
        cpu_baseline = dict(value=val, unit=UNIT, cores=O.num_threads(), kind="oracle",
                            sample=("oracle/fmm_oracle.cpp as it stands (fp64, OpenMP): full upward pass %.2f s + M2L/L2L/L2P/P2P for %d random leaves and "
                                    "their ancestors (%d of %d M2L pairs, %d particles) %.2f s; value = N / (t_up + t_down * pairs_total/pairs), i.e. %.0f s "
                                    "per full evaluate" % (t_up, int(mask.sum()), pairs, pairs_total, done, t_m - t_up, t_full)))

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3), ms_per_step=ms_per_step,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32" if esize == 4 else "f64", data="synthetic",
                config=dict(workload=args.workload, N=N, p=c["p"], s=c["s"], N_max=c["N_max"], theta=c["theta"], cross_level=args.cross_level,
                            outputs="potential+field",
                            L=info["L"], n_boxes=info["n_boxes"], n_weak=info["n_weak"], n_strong=info["n_strong"], n_p2p_pairs=info["n_p2p_pairs"],
                            l2="flushed between timed steps (512 MiB memset outside the event pairs)", parallelism="replicas x%d" % world,
                            schedule="concurrent: P2P, the tree passes (M2M, upper-level M2L, L2L) and the leaf-level M2L on three forked streams"),
                clocks=clocks, e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=N * esize, d2h_bytes_per_step=N * 4 * esize,
                                        ms_per_step=e2e_ms_max, steps=n_e2e),
                gpu_launches=launches * args.steps, gpu_launches_per_step=launches, roofline=roofline, stages=stages, plan_ms=plan_ms,
                alt_lists=alt, potential_only=pot_only, separate_targets=st_line, replan=replan, min_ms_per_step=float(step_ms.min()), wall_ms_per_step_incl_flush=t_wall * 1e3 / args.steps, cpu_baseline=cpu_baseline)
    print(json.dumps(line), flush=True)
    P.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2_cube1M_f32")
    ap.add_argument("--cpu-leaves", type=int, default=48, help="leaves in the cpu_baseline sample")
    ap.add_argument("--ref-leaves", type=int, default=16, help="leaves per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cross-level", type=int, default=0, choices=[0, 1],
                    help="interaction lists of the timed plan: 0 = same-level (paper default, PAPER.md:72-74), 1 = level marching (PAPER.md:82-89)")
    ap.add_argument("--no-alt-lists", action="store_true", help="skip the extra measurements (the other list kind; separate targets)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
