"""Evaluation pass at config-4 shape (m x 32, half the balls on the unit sphere and active, each with a multiplier row):
the input of `profiles/r2_config4_*.md`.  Run as a script it times `meb_eval_alm` with and without multiplier rows in
both precisions (CUDA events of the library, median of 5)."""
import sys

import numpy as np
import torch


def build(m, seed=1):
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    C = torch.randn((m, 32), dtype=torch.float64, device="cuda", generator=g)
    C /= C.norm(dim=1, keepdim=True)
    inner = torch.rand(m, device="cuda", generator=g) < 0.5
    C[inner] *= 0.5
    has = ~inner
    ns = int(has.sum())
    slot = torch.full((m,), -1, dtype=torch.int32, device="cuda")
    slot[has] = torch.arange(ns, dtype=torch.int32, device="cuda")
    U = torch.zeros(m, dtype=torch.float64, device="cuda"); U[has] = 1e-7
    V = 1e-7 * torch.randn((ns, 32), dtype=torch.float64, device="cuda", generator=g)
    x = torch.zeros(33, dtype=torch.float64, device="cuda"); x[0] = 0.999
    return C, U, slot, V, x, ns


def main():
    import os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import paper_2605_31425_b200.binding as meb
    m = int(sys.argv[1]) if len(sys.argv) > 1 else 10_000_000
    C64, U64, slot, V64, x, ns = build(m)
    for prec, dt in ((meb.MEB_FP64, torch.float64), (meb.MEB_FP32, torch.float32)):
        C, U, V = C64.to(dt), U64.to(dt), V64.to(dt)
        es = 8 if prec == meb.MEB_FP64 else 4
        with meb.Context(m, 32) as ctx:
            meb.meb_set_pass_timing(ctx, True)
            for name, (Uu, ss, VV) in (("no multiplier rows", (None, None, None)), ("%d multiplier rows" % ns, (U, slot, V))):
                ts = []
                for _ in range(6):
                    meb.meb_eval_alm(ctx, prec, C, None, Uu, ss, VV, x, x, 10.0, 1e-3)
                    ts.append(meb.meb_last_pass_info(ctx)[0])
                t = float(np.median(ts[1:]))
                nbytes = m * 32 * es + (0 if ss is None else m * (es + 4) + ns * 32 * es)
                print("%s, %s: %.4f ms, %.3f GB algorithmic, %.0f GB/s" % ("FP64" if es == 8 else "FP32", name, t, nbytes / 1e9,
                                                                           nbytes / t / 1e6), flush=True)


if __name__ == "__main__":
    main()
