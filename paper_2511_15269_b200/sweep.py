"""Scaling sweep of BASELINE.json config 5 (the paper's Figs. 5-10 shape): N x p x dtype x point set x N_max.

    python -m paper_2511_15269_b200.sweep [--out profiles/rNN_sweep.md] [--quick]

For every case: one plan (timed), 3 warm-up evaluates, then `--reps` evaluates timed with CUDA events around
`fmm_evaluate` (concurrent schedule, L2 flushed between evaluates by a 512 MiB memset outside the event pair); the
minimum and the mean are reported like the paper does, plus the serial per-stage times of
`fmm_evaluate_profiled`.  Inputs are the seeded synthetic sets of `inputs.py` (uniform cube, unit-sphere surface).
Argument marshalling and timing only; every step of the path runs in the CUDA library.
"""
import argparse
import itertools
import sys

import numpy as np
import torch

from . import fmm, inputs


def run_case(kind, N, dtype, p, N_max, s, theta, reps, flush):
    gen = inputs.uniform_cube if kind == "cube" else inputs.sphere_surface
    pos, q = gen(N, 50 + int(np.log10(N)), dtype)
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    d_pos = torch.from_numpy(pos).cuda()
    d_q = torch.from_numpy(q).cuda()
    P = fmm.Plan(d_pos, p, N_max, s, theta)
    info = P.info
    d_u = torch.empty(N, dtype=tdt, device="cuda")
    d_f = torch.empty((N, 3), dtype=tdt, device="cuda")
    for _ in range(3):
        fmm.fmm_evaluate(P.handle, d_q, d_u, d_f)
    ts = []
    for _ in range(reps):
        flush.zero_()
        a = torch.cuda.Event(enable_timing=True)
        b = torch.cuda.Event(enable_timing=True)
        a.record()
        fmm.fmm_evaluate(P.handle, d_q, d_u, d_f)
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    flush.zero_()
    st = fmm.fmm_evaluate_profiled(P.handle, d_q, d_u, d_f)
    ok = bool(torch.isfinite(d_u).all()) and bool(torch.isfinite(d_f).all())
    plan_ms = P.timings()["total"]
    P.close()
    del d_pos, d_q, d_u, d_f
    return dict(L=info["L"], n_weak=info["n_weak"], n_pairs=info["n_p2p_pairs"], min_ms=float(np.min(ts)), mean_ms=float(np.mean(ts)),
                plan_ms=plan_ms, m2l=st["m2l"], p2p=st["p2p"], rest=st["total"] - st["m2l"] - st["p2p"], finite=ok)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None, help="write the markdown table here (default: stdout)")
    ap.add_argument("--reps", type=int, default=10)
    ap.add_argument("--quick", action="store_true", help="N <= 1e6, N_max = 128 only")
    ap.add_argument("--theta", type=float, default=0.77)
    ap.add_argument("--sets", default="cube,sphere", help="comma list out of cube, sphere")
    ap.add_argument("--N", default=None, help="comma list of particle counts (default 1e4..1e7)")
    ap.add_argument("--p", default="4,8,12", help="comma list of orders")
    ap.add_argument("--dtype", default="float32,float64", help="comma list out of float32, float64")
    ap.add_argument("--nmax", default=None, help="comma list of N_max (default 32,128,512)")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        sys.exit("sweep needs a GPU")
    Ns = [10**4, 10**5, 10**6] + ([] if args.quick else [10**7])
    N_maxs = [128] if args.quick else [32, 128, 512]
    if args.N:
        Ns = [int(float(x)) for x in args.N.split(",")]
    if args.nmax:
        N_maxs = [int(x) for x in args.nmax.split(",")]
    ps = [int(x) for x in args.p.split(",")]
    dtypes = [dict(float32=np.float32, float64=np.float64)[x] for x in args.dtype.split(",")]
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    lines = ["| set | N | dtype | p | N_max | L | weak pairs | P2P pairs | plan ms | evaluate min ms | mean ms | Mparticles/s (min) | M2L ms | P2P ms | other ms |",
             "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    for kind, N, dtype, p, N_max in itertools.product(args.sets.split(","), Ns, dtypes, ps, N_maxs):
        try:
            r = run_case(kind, N, dtype, p, N_max, 3, args.theta, args.reps, flush)
        except Exception as e:  # report and go on: one failing case must not hide the others
            lines.append("| %s | %d | %s | %d | %d | failed: %s |" % (kind, N, np.dtype(dtype).name, p, N_max, str(e)[:80]))
            print(lines[-1], flush=True)
            continue
        lines.append("| %s | %d | %s | %d | %d | %d | %.3g | %.3g | %.1f | %.3f | %.3f | %.1f | %.3f | %.3f | %.3f |%s" % (
            kind, N, np.dtype(dtype).name, p, N_max, r["L"], r["n_weak"], r["n_pairs"], r["plan_ms"], r["min_ms"], r["mean_ms"],
            N / r["min_ms"] / 1e3, r["m2l"], r["p2p"], r["rest"], "" if r["finite"] else " non-finite output"))
        print(lines[-1], flush=True)
    if args.out:
        with open(args.out, "w") as f:
            f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
