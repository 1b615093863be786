#!/usr/bin/env python
"""bench.py -- time-to-solution of meb_solve and per-pass HBM GB/s on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--mode mixed|fp64] [--impl reference]
                    [--shard] [--no-extra] [--no-e2e] [--no-cpu-baseline]

A "step" is one whole meb_solve (one pass of the hot path: ingest, ALM evaluations, Newton solves,
multiplier updates, screening + compaction, feasibility check) on a seeded synthetic instance of a
BASELINE.json configuration.  BASELINE.json's metric quotes no configuration, so the N = 1 line is on the
LARGEST single-GPU one: configs[4] (m = 2e5 balls in R^10000, 16 GB of centres), mixed precision, which
exercises every row of SURVEY 8(a).  Prints ONE JSON line (see the task contract):

  value      seconds per solve with the balls already resident in HBM (CUDA events around K solves)
  e2e        the same through meb_solve_host with pinned HOST buffers (H2D inside the timed region)
  roofline   the dominant streaming kernel of the step.  `achieved` = algorithmic bytes per launch / launch
             duration from CUDA-EVENT pairs recorded on the launching stream around every streaming launch of
             one extra, host-stepped solve of the same instance (MEB_OPT_STEPPED: the same kernels, arguments
             and iterates as the graph-mode solves that are timed for `value`; inside a CUDA-graph WHILE node no
             event can be recorded per iteration).  `in_graph_globaltimer` is the same kernel's time inside the
             timed graph-mode solves from the %globaltimer stamps of its CTAs (last end - first start).
  configs    (N = 1) the other BASELINE.json configurations, FP64 and mixed, each with ms_per_step, the
             event-timed GB/s of every pass class and the solve statistics
  cpu_baseline  the CPU oracle timed on the host cores on a bounded sample (rank 0, N = 1)

N > 1 (torchrun): by default every rank solves its own seeded instance ("replicas"); with --shard the m balls
of ONE instance are partitioned over the ranks and the (d + O(10))-sized partial
reductions are all-gathered over NCCL at every reduction point.
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
HEADLINE_CONFIG = 5


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG, help="BASELINE.json configs[k-1], k = 1..5")
    ap.add_argument("--mode", default="mixed", choices=["mixed", "fp64"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--m", type=int, default=None, help="override m (debugging only; reported in config)")
    ap.add_argument("--cpu-sample", type=int, default=None, help="balls in the CPU-oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the per-config block (configs 1-5, both modes)")
    ap.add_argument("--shard", action="store_true", help="N > 1: partition the balls of one instance over the ranks")
    ap.add_argument("--paper-grid", action="store_true",
                    help="the paper's own deterministic instances (P:L289-299, grids of P:L319-320 and L335): one JSON "
                         "line with device times and the balls kept for the FP64 phase (Table 1, P:L326-333)")
    return ap.parse_args()


def workload_name(k, m, d, mode):
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


def oracle_time(C, R, mode):
    """Times oracle/ripalm.meb_solve, as it stands, on the given balls."""
    from oracle import ripalm
    t0 = time.perf_counter()
    c, r, info = ripalm.meb_solve(C, R, TOL, mode)
    return time.perf_counter() - t0, r, info


def cpu_threads():
    """Threads the oracle used: its elementwise numpy passes, which dominate, run on ONE thread (its few BLAS
    calls may use more, which is reported separately)."""
    return 1


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return int(max([p.get("num_threads", 1) for p in threadpool_info()] or [1]))
    except Exception:
        return 1


def cpu_baseline_entry(C, R, m, mode, dt, m_s):
    full = m_s >= m
    entry = {"value": dt * (m / m_s), "unit": UNIT, "cores": cpu_threads(), "kind": "oracle",
             "extrapolated": (not full), "measured_s": dt, "blas_threads_available": blas_threads(),
             "host_cores": os.cpu_count()}
    if full:
        entry["sample"] = f"the full instance ({m} balls), measured once; numpy oracle, elementwise passes on 1 thread"
    else:
        entry["sample"] = (f"first {m_s} of {m} balls of the same seeded instance: {dt:.3f} s measured, `value` is that "
                           f"times {m / m_s:.1f} (an EXTRAPOLATION: cost per pass is linear in m, the number of passes "
                           f"and |I_red| are not); the dense-V numpy oracle does not fit the full instance")
    return entry


def run_reference(args, rank, world):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only)."""
    import workloads
    if rank != 0:
        return
    k = args.config
    mf, d, _ = workloads.CONFIG_SHAPES[k]
    m = args.m or mf
    m_s = oracle_sample_size(k, m, d, args.cpu_sample)
    C, R = workloads.config(k, m_s, d)
    for _ in range(min(args.warmup, 1)):            # numpy needs no warm-up beyond the first import
        oracle_time(C[:min(m_s, 500)], None if R is None else R[:min(m_s, 500)], args.mode)
    times = []
    for _ in range(args.steps):
        dt, r, _info = oracle_time(C, R, args.mode)
        times.append(dt)
    per = sum(times) / len(times)
    entry = cpu_baseline_entry(C, R, m, args.mode, per, m_s)
    line = {"impl": "reference", "metric": METRIC, "value": entry["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": entry["value"] * 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(k, m, d, args.mode)},
            "cpu_baseline": entry,
            "e2e": {"value": entry["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------- B200 arm
def make_instance(k, m, d, seed, device, want_host):
    """Generates the seeded instance (threads over the independent 65,536-row blocks) and places it in HBM
    (row-major FP64 centres, FP64 radii or None).  With want_host the host copy is PINNED and returned (e2e leg)."""
    import numpy as np
    import torch
    import workloads
    has_r = workloads.CONFIG_SHAPES[k][2]
    dC = torch.empty((m, d), dtype=torch.float64, device=device)
    dR = torch.empty(m, dtype=torch.float64, device=device) if has_r else None
    hC = hR = None
    if want_host:
        hC = torch.empty((m, d), dtype=torch.float64, pin_memory=True)
        hR = torch.empty(m, dtype=torch.float64, pin_memory=True) if has_r else None
        workloads.config_into(k, hC.numpy(), None if hR is None else hR.numpy(), m, d, seed, threads=os.cpu_count() or 8)
        dC.copy_(hC)
        if dR is not None:
            dR.copy_(hR)
    else:
        lock = threading.Lock()

        def sink(row0, Cb, Rb):
            tC = torch.from_numpy(np.ascontiguousarray(Cb))
            with lock:                      # one stream of H2D copies; the draws of the other blocks overlap it
                dC[row0:row0 + Cb.shape[0]].copy_(tC)
                if dR is not None:
                    dR[row0:row0 + Cb.shape[0]].copy_(torch.from_numpy(np.ascontiguousarray(Rb)))
        workloads.config_into(k, None, None, m, d, seed, threads=min(os.cpu_count() or 8, 8), sink=sink)
    torch.cuda.synchronize()
    return dC, dR, hC, hR


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy test)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def ncu_traffic(cls_name, k):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, if one is recorded."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        with open(p) as f:
            return json.load(f).get(f"config{k}", {}).get(cls_name)
    except Exception:
        return None


def pass_table(meb, st_graph_list, st_step, peak):
    """Per pass class: event-timed launches of the stepped solve, and the in-graph globaltimer figure of the
    graph-mode solves."""
    names = {v: n for n, v in meb.PASS.items()}
    out = {}
    for i in range(8):
        n_ev = st_step["pass_ev_count"][i]
        n_g = sum(s["pass_count"][i] for s in st_graph_list)
        if n_ev == 0 and n_g == 0:
            continue
        e = {}
        if n_ev > 0:
            ms = st_step["pass_ev_ms"][i]
            by = st_step["pass_ev_bytes"][i]
            e.update({"launches_timed": n_ev, "ms_per_launch": ms / n_ev, "bytes_per_launch": by / n_ev,
                      "GBps": by / ms / 1e6 if ms > 0 else None,
                      "frac": (by / ms / 1e6 / peak) if (ms > 0 and i != meb.PASS["EVAL_REDUCED"]) else None})
        if n_g > 0:
            msg = sum(s["pass_ms"][i] for s in st_graph_list)
            byg = sum(s["pass_bytes"][i] for s in st_graph_list)
            e["in_graph_globaltimer"] = {"launches": n_g, "ms_per_launch": msg / n_g,
                                         "GBps": byg / msg / 1e6 if msg > 0 else None}
        out[names.get(i, str(i))] = e
    return out


def solve_summary(r, st):
    keys = ["outer_iters", "newton_iters", "cg_iters", "ag_iters", "passes_fp64_full", "passes_fp32_full", "passes_reduced",
            "passes_cut", "trials_skipped", "n_reduced", "rounds", "ms_phase_lo", "ms_phase_hi", "ms_check", "kkt",
            "delta_max", "n_support"]
    out = {"radius": r}
    out.update({k: st[k] for k in keys})
    return out


def bench_instance(meb, torch, ctx, dC, dR, mode, steps, warmup, timed, sampler_index):
    """Warm-up, K timed graph-mode solves (clocks sampled), then ONE host-stepped solve for the event times."""
    solve = lambda: meb.meb_solve(ctx, dC, dR, TOL, mode)
    for _ in range(max(warmup, 0)):
        solve()
    with ClockSampler(sampler_index) as clk:
        ms, wall, outs = timed(solve, steps)
    assert all(o[2]["converged"] == 1 for o in outs), "solve did not converge"
    meb.meb_set_option(ctx, meb.OPT["STEPPED"], True)
    try:
        cs, rs, st_step = meb.meb_solve(ctx, dC, dR, TOL, mode)
    finally:
        meb.meb_set_option(ctx, meb.OPT["STEPPED"], False)
    c, r, st = outs[-1]
    assert rs == r and torch.equal(cs, c), "the stepped solve must reproduce the graph-mode solve bit for bit"
    return ms, wall, outs, st_step, clk.summary()


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
    if args.shard and world > 1:
        from paper_2605_31425_b200 import shard as meb_shard
        return meb_shard.bench_sharded(args, rank, world, local_rank, METRIC, UNIT, TOL, workload_name)
    k = args.config
    mf, d, _ = workloads.CONFIG_SHAPES[k]
    m = args.m or mf
    mode = meb.MEB_MODE_MIXED if args.mode == "mixed" else meb.MEB_MODE_FP64
    want_e2e = not args.no_e2e
    dC, dR, hC, hR = make_instance(k, m, d, rank, device, want_e2e)   # seed = rank: replicas solve different instances
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

    ms, wall, outs, st_step, clocks = bench_instance(meb, torch, ctx, dC, dR, mode, args.steps, args.warmup, timed,
                                                     local_rank)
    c, r, st = outs[-1]

    # ---- roofline of the dominant streaming kernel: CUDA-event pairs of the stepped solve
    peak, peak_src = measured_peak()
    per_pass = pass_table(meb, [o[2] for o in outs], st_step, peak)
    names = {v: n for n, v in meb.PASS.items()}
    hbm = [i for i in range(8) if i != meb.PASS["EVAL_REDUCED"] and st_step["pass_ev_count"][i] > 0]
    dom = max(hbm, key=lambda i: st_step["pass_ev_ms"][i])
    pd = per_pass[names[dom]]
    n_graph_dom = sum(o[2]["pass_count"][dom] for o in outs) or (st_step["pass_ev_count"][dom] * len(outs))
    roofline = {"bound": "hbm", "kernel": names[dom], "achieved": pd["GBps"], "peak": peak, "unit": "GB/s",
                "frac": pd["GBps"] / peak, "frac_of_8TBps_nominal": pd["GBps"] / 8000.0, "peak_source": peak_src,
                "timing": "CUDA events around each launch of a host-stepped solve of the same instance",
                "traffic": ncu_traffic(names[dom], k),
                "algorithmic_bytes_per_launch": pd["bytes_per_launch"], "ms_per_launch": pd["ms_per_launch"],
                "share_of_step": n_graph_dom * pd["ms_per_launch"] / ms,
                "in_graph_globaltimer": pd.get("in_graph_globaltimer"), "per_pass": per_pass}

    # ---- end to end: host buffers in, (r, c) out, through meb_solve_host
    e2e = None
    if want_e2e:
        solve_h = lambda: meb.meb_solve_host(ctx, hC, hR, TOL, mode)
        solve_h()
        e2e_steps = args.steps if hC.numel() * 8 < (2 << 30) else min(args.steps, 3)
        ms_h, wall_h, outs_h = timed(solve_h, e2e_steps)
        e2e = {"value": ms_h / 1e3 / e2e_steps, "unit": UNIT, "steps": e2e_steps,
               "h2d_bytes_per_step": int(hC.numel() * 8 + (0 if hR is None else hR.numel() * 8)),
               "d2h_bytes_per_step": int((d + 1) * 8), "wall_s_per_step": wall_h / e2e_steps,
               "note": "PCIe-bound: one host-to-device copy of the centres, then the device-resident solve"}

    line = {"metric": METRIC, "value": ms / 1e3 / args.steps, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": workload_name(k, m, d, args.mode), "multi_gpu": "replicas only" if world > 1 else "single GPU",
                       "l2": "inputs larger than L2 (%.0f MB streamed per pass)" % (pd["bytes_per_launch"] / 1e6)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(sum(o[2]["kernel_launches"] for o in outs)),
            "roofline": roofline, "wall_s_per_step": wall / args.steps, "solve": solve_summary(r, st)}

    # ---- CPU oracle on the host cores (rank 0, N = 1): bounded sample of the headline instance
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        m_s = oracle_sample_size(k, m, d, args.cpu_sample)
        if hC is not None:
            Cs, Rs = hC.numpy()[:m_s], (None if hR is None else hR.numpy()[:m_s])
        else:
            Cs, Rs = workloads.config(k, m_s, d, rank)
        dt, r_o, _ = oracle_time(Cs, Rs, args.mode)
        line["cpu_baseline"] = cpu_baseline_entry(Cs, Rs, m, args.mode, dt, m_s)
    # ---- the other configurations (N = 1): FP64 and mixed, event-timed passes, solve statistics
    extras = world == 1 and not args.no_extra and args.m is None
    block = {}

    def extra(kk, mk, dk, ectx, eC, eR, mname):
        mmode = meb.MEB_MODE_FP64 if mname == "fp64" else meb.MEB_MODE_MIXED
        nst = 20 if kk <= 2 else 5
        ems, ewall, eouts, est_step, eclk = bench_instance(meb, torch, ectx, eC, eR, mmode, nst, 2, timed, local_rank)
        ec, er, est = eouts[-1]
        block[f"config{kk}_{mname}"] = {
            "workload": workload_name(kk, mk, dk, mname), "steps": nst, "ms_per_step": ems / nst,
            "per_pass": pass_table(meb, [o[2] for o in eouts], est_step, peak), "clocks": eclk,
            "solve": solve_summary(er, est)}

    if extras:
        extra(k, m, d, ctx, dC, dR, "fp64" if args.mode == "mixed" else "mixed")
    ctx.close()
    del dC, dR, hC, hR, ctx
    torch.cuda.empty_cache()
    if extras:
        for kk in (1, 2, 3, 4, 5):
            if kk == k:
                continue
            mk, dk, _ = workloads.CONFIG_SHAPES[kk]
            eC, eR, _, _ = make_instance(kk, mk, dk, 0, device, False)
            ectx = meb.Context(mk, dk)
            for mname in ("fp64", "mixed"):
                extra(kk, mk, dk, ectx, eC, eR, mname)
            if kk == 2 and rank == 0 and not args.no_cpu_baseline:
                # the oracle on the FULL config-2 instance, measured once (about a minute on one core)
                Ch = eC.cpu().numpy()
                dt2, r2, _ = oracle_time(Ch, None, "mixed")
                block["config2_mixed"]["cpu_oracle"] = cpu_baseline_entry(Ch, None, mk, "mixed", dt2, mk)
                block["config2_mixed"]["cpu_oracle"]["radius"] = r2
                del Ch
            ectx.close()
            del eC, eR, ectx
            torch.cuda.empty_cache()
        line["configs"] = block
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_paper_grid():
    """The paper's own workload: d in {20,30,40,50} x m in {1e3..1e5} (Table 1) and
    d in {1e2..1e4} x m in {1e3, 5e3}.  Device time of the FP64 and of the mixed solve (best of 3), the
    number of balls kept for phase 2 and the radius."""
    import torch
    import paper_2605_31425_b200 as meb
    import workloads
    rows = []
    grid = [(d, m) for d in (20, 30, 40, 50) for m in (1000, 5000, 10000, 50000, 100000)]
    grid += [(d, m) for d in (100, 500, 1000, 5000, 10000) for m in (1000, 5000)]
    for d, m in grid:
        C, R = workloads.paper_instance(m, d)
        dC, dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
        rec = {"d": d, "m": m}
        with meb.Context(m, d) as ctx:
            for mode, name in ((meb.MEB_MODE_FP64, "fp64"), (meb.MEB_MODE_MIXED, "mixed")):
                best = None
                for _ in range(3):
                    c, r, st = meb.meb_solve(ctx, dC, dR, TOL, mode, allow_not_converged=True)
                    best = st["ms_total"] if best is None else min(best, st["ms_total"])
                rec[name + "_ms"] = best
                rec[name + "_converged"] = st["converged"]
                rec[name + "_radius"] = r
                if name == "mixed":
                    rec["kept"] = st["n_reduced"]
        rows.append(rec)
    print(json.dumps({"workload": "paper instances (LCG generator, P:L289-299)", "tol": TOL, "rows": rows}), flush=True)


def main():
    args = parse_args()
    if args.paper_grid:
        return run_paper_grid()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_b200(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
