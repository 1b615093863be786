#!/usr/bin/env python
"""bench.py -- time-to-solution of meb_solve and per-pass HBM GB/s on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--mode mixed|fp64] [--impl reference]

A "step" is one whole meb_solve (one pass of the hot path: ingest, ALM evaluations, Newton solves,
multiplier updates, screening + compaction, feasibility check) on a seeded synthetic instance of the
BASELINE.json configuration (default: configs[1], m = 1e6 points in R^100, mixed precision, which
exercises every row of SURVEY 8(a)).  Prints ONE JSON line (see the task contract):

  value      seconds per solve with the balls already resident in HBM (CUDA events around K solves)
  e2e        the same through meb_solve_host with pinned HOST buffers (H2D inside the timed region)
  roofline   the dominant streaming kernel of the step: algorithmic bytes / launch duration measured
             INSIDE the timed solves (evaluation passes run inside a CUDA-graph WHILE node, where no
             event can be recorded per iteration: their device time comes from %globaltimer stamps of
             the kernel's CTAs; ingest / screen / feasibility launches are bracketed by CUDA events),
             plus `events_check`: the same kernel timed stand-alone with CUDA events
  cpu_baseline  the CPU oracle timed on the host cores on a bounded sample (rank 0, N = 1)

N > 1 (torchrun): the path does not shard in this round ("replicas only"): every rank
solves its own seeded instance, time = max over ranks, value = time per solve of the whole job.
--impl reference: the oracle (oracle/ripalm.py) as it stands, on the host cores, bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "meb_solve_time_to_1e-8_rel_kkt"
UNIT = "s"
TOL = 1e-8


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[k-1], k = 1..5")
    ap.add_argument("--mode", default="mixed", choices=["mixed", "fp64"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--m", type=int, default=None, help="override m (debugging only; reported in config)")
    ap.add_argument("--cpu-sample", type=int, default=None, help="balls in the CPU-oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload_name(k, m, d, mode):
    import workloads
    mf, df, has_r = workloads.CONFIG_SHAPES[k]
    kind = {1: "balls N(0,1), r~U[0,0.1]", 2: "points N(0,1)", 3: "balls U[-1,1]^d, r~U[0,1]",
            4: "boundary-heavy points", 5: "anisotropic balls, r~lognormal(-3,1)"}[k]
    return f"config{k}: {kind}, m={m}, d={d}, {mode}, tol=1e-8, seed 0"


# ------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs (one long-lived
    `nvidia-smi -lms` process: spawning one per sample is slower than a short timed region)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.proc = None
        self.th = None

    def _run(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.strip().split(",")])

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._run, daemon=True)
            self.th.start()
            time.sleep(0.3)                      # let the first samples arrive before the region starts
            self.rows.clear()
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.06)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.th.join(timeout=5)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                   r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------- oracle arm
def oracle_sample_size(k, m, d, override=None):
    """Balls in the bounded CPU sample: about 10-30 s of oracle work per solve (calibrated: the numpy
    oracle needs ~1.3e-6 s per ball-coordinate per mixed solve on one Xeon core)."""
    if override:
        return min(m, int(override))
    budget_elems = 8_000_000            # m_s * d
    return max(256, min(m, budget_elems // max(d, 1)))


def oracle_solve_sample(k, m, d, mode, m_s):
    """Times oracle/ripalm.meb_solve on the first m_s balls of the workload (a prefix of the same
    seeded instance; config 4 re-draws its sphere/interior permutation at size m_s)."""
    import numpy as np  # noqa: F401
    import workloads
    from oracle import ripalm
    C, R = workloads.config(k, m_s, d)
    t0 = time.perf_counter()
    c, r, info = ripalm.meb_solve(C, R, TOL, mode)
    dt = time.perf_counter() - t0
    return dt, r, info


def cpu_threads():
    """Threads available to the oracle's numpy (its BLAS calls may use them; its elementwise passes,
    which dominate, run on one thread)."""
    try:
        from threadpoolctl import threadpool_info
        n = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
        return int(n)
    except Exception:
        return 1


def run_reference(args, rank, world):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only)."""
    import workloads
    if rank != 0:
        return
    k = args.config
    mf, d, _ = workloads.CONFIG_SHAPES[k]
    m = args.m or mf
    m_s = oracle_sample_size(k, m, d, args.cpu_sample)
    for _ in range(min(args.warmup, 1)):            # numpy needs no warm-up beyond the first import
        oracle_solve_sample(k, m, d, args.mode, min(m_s, 2000))
    times = []
    for _ in range(args.steps):
        dt, r, _info = oracle_solve_sample(k, m, d, args.mode, m_s)
        times.append(dt)
    per = sum(times) / len(times)
    scaled = per * (m / m_s)
    sample = (f"first {m_s} of {m} balls of the same seeded instance, {per:.3f} s per solve measured, "
              f"scaled x{m / m_s:.1f} to m (cost per pass is linear in m); numpy: elementwise passes on 1 thread, "
              f"BLAS calls on up to `cores` threads")
    line = {"impl": "reference", "metric": METRIC, "value": scaled, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": scaled * 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(k, m, d, args.mode)},
            "cpu_baseline": {"value": scaled, "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": scaled, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------- B200 arm
def upload_instance(k, m, d, seed, device):
    """Generates the seeded instance block by block on the host and places it in HBM (row-major FP64
    centres, FP64 radii or None).  Also returns pinned host copies when they fit (for the e2e leg)."""
    import numpy as np
    import torch
    import workloads
    has_r = workloads.CONFIG_SHAPES[k][2]
    dC = torch.empty((m, d), dtype=torch.float64, device=device)
    dR = torch.empty(m, dtype=torch.float64, device=device) if has_r else None
    for row0, Cb, Rb in workloads.config_blocks(k, m, d, seed):
        n = Cb.shape[0]
        dC[row0:row0 + n].copy_(torch.from_numpy(np.ascontiguousarray(Cb)))
        if dR is not None:
            dR[row0:row0 + n].copy_(torch.from_numpy(np.ascontiguousarray(Rb)))
    return dC, dR


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy test)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def ncu_traffic(cls_name, k, mode):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, if one is recorded."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        with open(p) as f:
            return json.load(f).get(f"config{k}", {}).get(cls_name)
    except Exception:
        return None


def run_b200(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_2605_31425_b200 as meb
    import workloads

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    k = args.config
    mf, d, _ = workloads.CONFIG_SHAPES[k]
    m = args.m or mf
    mode = meb.MEB_MODE_MIXED if args.mode == "mixed" else meb.MEB_MODE_FP64
    dC, dR = upload_instance(k, m, d, rank, device)       # seed = rank: replicas solve different instances
    ctx = meb.Context(m, d)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        outs = [fn() for _ in range(steps)]
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        ms = max(e0.elapsed_time(e1), 0.0)
        barrier()
        if world > 1:
            t = torch.tensor([ms, wall * 1e3], dtype=torch.float64, device=device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms, wall = float(t[0]), float(t[1]) / 1e3
        return ms, wall, outs

    solve = lambda: meb.meb_solve(ctx, dC, dR, TOL, mode)
    for _ in range(max(args.warmup, 0)):
        solve()
    with ClockSampler(local_rank) as clk:
        ms, wall, outs = timed(solve, args.steps)
    clocks = clk.summary()
    c, r, st = outs[-1]
    assert all(o[2]["converged"] == 1 for o in outs), "solve did not converge"

    # ---- roofline of the dominant streaming kernel, from the event pairs recorded inside the timed solves
    names = {v: n for n, v in meb.PASS.items()}
    tot_ms = [sum(o[2]["pass_ms"][i] for o in outs) for i in range(8)]
    tot_by = [sum(o[2]["pass_bytes"][i] for o in outs) for i in range(8)]
    tot_n = [sum(o[2]["pass_count"][i] for o in outs) for i in range(8)]
    hbm_classes = [i for i in range(8) if i != meb.PASS["EVAL_REDUCED"] and tot_n[i] > 0]
    dom = max(hbm_classes, key=lambda i: tot_ms[i])
    peak, peak_src = measured_peak()
    per_pass = {names.get(i, str(i)): {"launches": tot_n[i], "ms_per_launch": tot_ms[i] / tot_n[i],
                                       "GBps": tot_by[i] / tot_ms[i] / 1e6 if tot_ms[i] > 0 else None,
                                       "bytes_per_launch": tot_by[i] / tot_n[i]}
                for i in range(8) if tot_n[i] > 0}
    ach = tot_by[dom] / tot_ms[dom] / 1e6
    roofline = {"bound": "hbm", "kernel": names[dom], "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak, "frac_of_8TBps_nominal": ach / 8000.0, "peak_source": peak_src,
                "traffic": ncu_traffic(names[dom], k, args.mode),
                "algorithmic_bytes_per_launch": tot_by[dom] / tot_n[dom],
                "share_of_step": tot_ms[dom] / ms, "per_pass": per_pass}

    # ---- cross-check: the dominant evaluation kernel alone, CUDA events around each launch
    try:
        import numpy as np
        reps = 10
        if args.mode == "mixed":
            ing = meb.meb_ingest(ctx, dC, dR, 1024, want_shadow=True)
            Cp, Rp, prec = ing["C32"], ing["R32"], meb.MEB_FP32
            x0 = torch.zeros(d + 1, dtype=torch.float64, device=device); x0[0] = 0.9 * ing["L"]
        else:
            ing = meb.meb_ingest(ctx, dC, dR, 1024)
            Cp, Rp, prec = dC, dR, meb.MEB_FP64
            x0 = torch.cat([torch.tensor([0.9 * ing["L"]], dtype=torch.float64, device=device), ing["c0"]])
        meb.meb_set_pass_timing(ctx, True)
        tms = []
        for _ in range(reps + 2):
            meb.meb_eval_alm(ctx, prec, Cp, Rp, None, None, None, x0, x0, 1.0 / ing["L"], 1.0 / ing["L"] ** 2)
            tms.append(meb.meb_last_pass_info(ctx))
        meb.meb_set_pass_timing(ctx, False)
        tms = tms[2:]
        ev_ms = sum(t[0] for t in tms) / len(tms)
        roofline["events_check"] = {"kernel": "eval_alm stand-alone (no multipliers), CUDA events",
                                    "ms_per_launch": ev_ms, "GBps": tms[0][1] / ev_ms / 1e6,
                                    "bytes_per_launch": tms[0][1]}
        del ing, Cp, Rp
    except Exception as exc:  # the cross-check must never take the bench line down
        roofline["events_check"] = {"error": repr(exc)}

    # ---- end to end: host buffers in, (r, c) out, through meb_solve_host
    e2e = None
    if not args.no_e2e:
        hC = dC.cpu().pin_memory()
        hR = None if dR is None else dR.cpu().pin_memory()
        solve_h = lambda: meb.meb_solve_host(ctx, hC, hR, TOL, mode)
        solve_h()
        ms_h, wall_h, outs_h = timed(solve_h, args.steps)
        e2e = {"value": ms_h / 1e3 / args.steps, "unit": UNIT,
               "h2d_bytes_per_step": int(hC.numel() * 8 + (0 if hR is None else hR.numel() * 8)),
               "d2h_bytes_per_step": int((d + 1) * 8), "wall_s_per_step": wall_h / args.steps}
        del hC, hR

    line = {"metric": METRIC, "value": ms / 1e3 / args.steps, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": workload_name(k, m, d, args.mode), "multi_gpu": "replicas only",
                       "l2": "inputs larger than L2 (%.0f MB streamed per pass)" % (tot_by[dom] / tot_n[dom] / 1e6)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(sum(o[2]["kernel_launches"] for o in outs)),
            "roofline": roofline, "wall_s_per_step": wall / args.steps,
            "solve": {"radius": r, "kkt": st["kkt"], "delta_max": st["delta_max"],
                      "outer_iters": st["outer_iters"], "newton_iters": st["newton_iters"],
                      "cg_iters": st["cg_iters"], "passes_fp64_full": st["passes_fp64_full"],
                      "passes_fp32_full": st["passes_fp32_full"], "passes_reduced": st["passes_reduced"], "passes_cut": st["passes_cut"],
                      "n_reduced": st["n_reduced"], "rounds": st["rounds"],
                      "ms_phase_lo": st["ms_phase_lo"], "ms_phase_hi": st["ms_phase_hi"],
                      "ms_check": st["ms_check"]}}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        m_s = oracle_sample_size(k, m, d, args.cpu_sample)
        dt, r_o, _ = oracle_solve_sample(k, m, d, args.mode, m_s)
        line["cpu_baseline"] = {"value": dt * (m / m_s), "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
                                "sample": f"first {m_s} of {m} balls of the same seeded instance: {dt:.3f} s "
                                          f"measured, scaled x{m / m_s:.1f} (cost per pass is linear in m); numpy: elementwise "
                                          f"passes on 1 thread, BLAS calls on up to `cores` threads"}
    ctx.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_b200(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
