"""Multi-GPU plumbing of the sharded solve: one process per GPU, the m balls of ONE
instance partitioned into contiguous row blocks, `torch.distributed` for the all-gather of the ranks' partial
records.  Marshalling only: every arithmetic step, including the rank-ordered addition of the gathered records,
runs in the kernels of libmeb_b200.so (``meb_solve_sharded``, csrc/meb_shard.cu).

* ``partition(m, nranks)``        contiguous, balanced row blocks: rank r owns [floor(r m / N), floor((r+1) m / N))
* ``gather_records(x, group)``    rank-ordered all-gather of a fixed-size record (any backend: NCCL on GPUs, gloo on CPU)
* ``globalize(idx, row_offset)``  local int32 indices of a rank -> global indices (index sets concatenate in rank order)
* ``solve_sharded(...)``          the solve of this rank's block, NCCL all-gather as the exchange
* ``ThreadRanks``                 N ranks as N host threads of ONE process sharing one GPU (tests on a single GPU): the
                                  exchange is a host-side barrier plus device copies; no kernel waits for another
"""
from __future__ import annotations

import threading

import torch

from . import binding as meb


def partition(m: int, nranks: int):
    """[(row_offset, m_local)] for ranks 0..nranks-1: contiguous, sizes differ by at most one, in rank order."""
    bounds = [(r * m) // nranks for r in range(nranks + 1)]
    return [(bounds[r], bounds[r + 1] - bounds[r]) for r in range(nranks)]


def gather_records(local: torch.Tensor, group=None) -> torch.Tensor:
    """All-gather of one fixed-size record per rank; row r of the result is rank r's record (rank order)."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    out = torch.empty((world,) + tuple(local.shape), dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(out.view(-1), local.contiguous().view(-1), group=group)
    return out


def globalize(local_idx: torch.Tensor, row_offset: int) -> torch.Tensor:
    """Global ball indices of a rank's local index list (int64: m_global may exceed what int32 holds per rank)."""
    return local_idx.to(torch.int64) + int(row_offset)


class _Exchange:
    """Send / receive records of one rank and the all-gather callable handed to ``meb_solve_sharded``."""

    def __init__(self, d: int, nranks: int, device):
        n = meb.meb_shard_record_doubles(d)
        self.send = torch.zeros(n, dtype=torch.float64, device=device)
        self.recv = torch.zeros(n * nranks, dtype=torch.float64, device=device)
        self.nranks = nranks


def solve_sharded(ctx, centers_local, radii_local, row_offset, m_global, tol=1e-8,
                  precision_mode=meb.MEB_MODE_MIXED, params=None, group=None, allow_not_converged=False):
    """Solve with this process's row block; ``torch.distributed`` (NCCL) must be initialised.  The context must
    have been created on the current stream (the all-gather is ordered on it)."""
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    ex = _Exchange(centers_local.shape[1], world, centers_local.device)

    def allgather(n):
        dist.all_gather_into_tensor(ex.recv[:n * world], ex.send[:n], group=group)
        return 0

    return meb.meb_solve_sharded(ctx, rank, world, centers_local, radii_local, row_offset, m_global, ex.send, ex.recv,
                                 allgather, tol, precision_mode, params, allow_not_converged)


class ThreadRanks:
    """N ranks emulated by N host threads of one process on ONE GPU.  Every thread owns a context on its own
    stream and its block of rows; the exchange synchronises the thread's stream, meets the others at a host
    barrier, copies all send records into its receive buffer (device copies on its stream) and meets them again
    before anyone overwrites a send record.  Kernels never wait on kernels, so this is safe on a single device."""

    def __init__(self, nranks: int):
        self.n = nranks
        self.barrier = threading.Barrier(nranks)
        self.ex = [None] * nranks
        self.results = [None] * nranks
        self.errors = [None] * nranks

    def _run(self, r, C, R, parts, m_global, tol, mode, params, device):
        try:
            torch.cuda.set_device(device)
            stream = torch.cuda.Stream(device=device)
            with torch.cuda.stream(stream):
                off, ml = parts[r]
                Cl = C[off:off + ml].contiguous()
                Rl = None if R is None else R[off:off + ml].contiguous()
                d = C.shape[1]
                self.ex[r] = _Exchange(d, self.n, device)
                ctx = meb.Context(ml, d, stream=stream)
                stream.synchronize()
                self.barrier.wait()

                def allgather(n):
                    try:
                        stream.synchronize()
                        self.barrier.wait()
                        mine = self.ex[r]
                        with torch.cuda.stream(stream):
                            for q in range(self.n):
                                mine.recv[q * n:(q + 1) * n].copy_(self.ex[q].send[:n])
                        stream.synchronize()
                        self.barrier.wait()
                        return 0
                    except threading.BrokenBarrierError:
                        return 1                      # another rank failed: the library returns an error here too

                self.results[r] = meb.meb_solve_sharded(ctx, r, self.n, Cl, Rl, off, m_global, self.ex[r].send,
                                                        self.ex[r].recv, allgather, tol, mode, params, True)
                ctx.close()
        except BaseException as exc:      # noqa: BLE001 -- reported to the caller; the barrier is broken for the others
            self.errors[r] = exc
            self.barrier.abort()

    def solve(self, C, R, tol=1e-8, mode=meb.MEB_MODE_MIXED, params=None):
        """C (m, d) / R (m,) CUDA float64 tensors of the WHOLE instance; returns [(c, r, stats)] per rank."""
        device = C.device
        m = C.shape[0]
        parts = partition(m, self.n)
        torch.cuda.synchronize()
        ths = [threading.Thread(target=self._run, args=(r, C, R, parts, m, tol, mode, params, device)) for r in range(self.n)]
        for t in ths:
            t.start()
        for t in ths:
            t.join()
        for e in self.errors:
            if e is not None and not isinstance(e, threading.BrokenBarrierError):
                raise e
        for e in self.errors:
            if e is not None:
                raise e
        return self.results


def bench_sharded(args, rank, world, local_rank, metric, unit, tol, workload_name):
    """bench.py --gpus N --shard: ONE instance of the configuration, its balls partitioned over the N ranks."""
    import json
    import time

    import numpy as np
    import torch.distributed as dist

    import workloads
    device = torch.device("cuda", local_rank)
    k = args.config
    mf, d, has_r = workloads.CONFIG_SHAPES[k]
    m = args.m or mf
    off, ml = partition(m, world)[rank]
    mode = meb.MEB_MODE_MIXED if args.mode == "mixed" else meb.MEB_MODE_FP64
    # this rank's rows of the global seeded instance: the 65,536-row blocks that overlap [off, off + ml)
    Cl = torch.empty((ml, d), dtype=torch.float64, device=device)
    Rl = torch.empty(ml, dtype=torch.float64, device=device) if has_r else None
    for row0, Cb, Rb in workloads.config_blocks(k, m, d, 0):
        lo, hi = max(row0, off), min(row0 + Cb.shape[0], off + ml)
        if lo < hi:
            Cl[lo - off:hi - off].copy_(torch.from_numpy(np.ascontiguousarray(Cb[lo - row0:hi - row0])))
            if Rl is not None:
                Rl[lo - off:hi - off].copy_(torch.from_numpy(np.ascontiguousarray(Rb[lo - row0:hi - row0])))
    ctx = meb.Context(ml, d)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    solve = lambda: solve_sharded(ctx, Cl, Rl, off, m, tol, mode)
    for _ in range(max(args.warmup, 0)):
        solve()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    outs = [solve() for _ in range(args.steps)]
    e1.record()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    t = torch.tensor([e0.elapsed_time(e1), wall * 1e3], dtype=torch.float64, device=device)
    barrier()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t[0])
    c, r, st = outs[-1]
    line = {"metric": metric, "value": ms / 1e3 / args.steps, "unit": unit, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": False, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(k, m, d, args.mode), "multi_gpu": f"sharded by balls over {world} ranks",
                       "exchange": "NCCL all-gather of (d + 16) doubles per evaluation, rank-ordered sums"},
            "gpu_launches": int(sum(o[2]["kernel_launches"] for o in outs)),
            "solve": {"radius": r, "converged": st["converged"], "passes_fp64_full": st["passes_fp64_full"],
                      "passes_fp32_full": st["passes_fp32_full"], "n_reduced_local": st["n_reduced"]},
            "e2e": None, "wall_s_per_step": float(t[1]) / 1e3 / args.steps}
    ctx.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    dist.destroy_process_group()
