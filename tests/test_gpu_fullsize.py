"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (config 2:
m = 1e6 points in R^100, mixed precision; run with -m gpu).

* whole solve: the returned ball is feasible to 1e-10 (1 + r) (checked on the host over all m), and its
  radius is within 1e-8 of the optimum by a two-sided argument that needs no full-size oracle run:
  MEB(subset) <= MEB(all) <= r_gpu for ANY subset, and the oracle (run to 1e-10) on the balls within
  2% of the returned boundary gives MEB(subset); r_gpu <= (1 + 1e-8) MEB(subset) closes the sandwich.
* eval_alm (FP32, the dominant kernel of the bench): per-ball outputs of sampled balls against the
  oracle evaluated one ball at a time, and the reductions against the oracle's full pass.
"""
import numpy as np
import pytest
import torch

import workloads
from oracle import primitives as prim
from oracle import ripalm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    meb.load()
    return meb


@pytest.fixture(scope="module")
def config2():
    C, R = workloads.config(2)                      # 1e6 x 100, points
    return C, torch.from_numpy(C).cuda()


def test_full_size_mixed_solve_sandwich(meb, config2):
    C, dC = config2
    m, d = C.shape
    with meb.Context(m, d) as ctx:
        c, r, st = meb.meb_solve(ctx, dC, None, 1e-8, meb.MEB_MODE_MIXED)
    c = c.numpy()
    assert st["converged"] == 1 and st["passes_fp32_full"] > 0 and st["rounds"] >= 1
    dist = np.sqrt(((C - c[None, :]) ** 2).sum(axis=1))
    assert dist.max() - r <= 1e-10 * (1 + r)                       # feasible for ALL m balls
    near = np.flatnonzero(dist >= 0.98 * r)                        # a subset that contains the support
    assert 0 < near.size < 5000
    cs, rs, info = ripalm.meb_solve(C[near], None, 1e-10, "fp64")
    assert info["converged"]
    assert rs <= r * (1 + 1e-12)                                   # MEB(subset) <= MEB(all) <= r
    assert r - rs <= 1e-8 * rs                                     # ... and r is within 1e-8 of it
    assert np.linalg.norm(c - cs) <= 1e-5 * (1 + rs)


def test_full_size_eval_fp32_sampled_and_reduced(meb, config2):
    C, dC = config2
    m, d = C.shape
    rng = np.random.default_rng(3)
    with meb.Context(m, d) as ctx:
        ing = meb.meb_ingest(ctx, dC, None, 1024, want_shadow=True)
        C32 = ing["C32"]
        L = ing["L"]
        x = np.concatenate([[0.93 * L], 0.01 * rng.standard_normal(d)])     # generic point, ~2% of the balls active
        xd = torch.from_numpy(x).cuda()
        sigma, tau = 1.0 / L, 1.0 / L ** 2
        res = meb.meb_eval_alm(ctx, meb.MEB_FP32, C32, None, None, None, None, xd, xd, sigma, tau, per_ball=True)
        s = res["scalars"].cpu().numpy()
        g = res["grad"].cpu().numpy()
        t_gpu = res["t"].cpu().numpy()
        lam_gpu = res["lam"].cpu().numpy()
    Ch = C32.cpu().numpy().astype(np.float64)                      # the very floats the kernel read
    zero = np.zeros(m)
    ev = prim.eval_alm(Ch, None, zero, np.zeros((m, d), dtype=np.float32), x, x, sigma, tau, dtype=np.float32)
    a, nb = ev["a"].astype(np.float64), ev["nb"].astype(np.float64)
    mag = np.abs(a) + nb
    near = (np.abs(nb - a) <= 1e-4 * mag) | (np.abs(nb + a) <= 1e-4 * mag)
    # sampled balls, one by one
    for i in rng.choice(m, 2000, replace=False):
        if near[i]:
            continue
        one = prim.eval_alm(Ch[i:i + 1], None, zero[:1], np.zeros((1, d), dtype=np.float32), x, x, sigma, tau,
                            dtype=np.float32)
        assert abs(t_gpu[i] - float(one["t"][0])) <= 1e-5 * mag[i]
        assert abs(lam_gpu[i] - float(one["lam"][0])) <= 4e-5
    # reductions of the whole pass, relative to the sums of |terms|
    E = meb.EV
    slack = near.sum() * 4.0 * float(mag.max()) ** 2 * sigma
    assert abs(s[E["SUM_PROJ2"]] - ev["sum_proj2"]) <= 1e-5 * ev["scale_proj2"] + slack
    assert abs(s[E["SUM_UPLUS"]] - ev["sum_uplus"]) <= 1e-5 * ev["scale_uplus"] + slack
    gscale = np.concatenate([[1 + ev["scale_uplus"]], ev["scale_vplus"]])
    assert np.linalg.norm(g - ev["grad"]) <= 1e-5 * np.linalg.norm(gscale) + slack
    if not near.any():
        assert int(s[E["N_B3"]]) == ev["n_b3"] and int(s[E["N_B1"]]) == ev["n_b1"]
