"""Sharded solve on ONE GPU: the N ranks are N host threads of this process, each with
its own context, stream and block of rows (paper_2605_31425_b200.shard.ThreadRanks); the exchange is a host barrier
plus device copies, so no kernel ever waits for another one.  Checks: every rank returns the SAME bits (replicated
controllers on rank-ordered sums), the radius matches the oracle, the ball is feasible for ALL m balls."""
import numpy as np
import pytest
import torch

import workloads
from oracle import ripalm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    meb.load()
    return meb


def _violation(C, R, c, r):
    return float(np.max(np.sqrt(((C - c) ** 2).sum(1)) + (0 if R is None else R) - r))


@pytest.mark.parametrize("mode", ["fp64", "mixed"])
@pytest.mark.parametrize("k,m,d,nranks", [(1, 6_001, 10, 2), (2, 20_000, 100, 3), (3, 2_000, 1000, 2), (4, 30_000, 32, 2)])
def test_sharded_solve_matches_oracle(meb, k, m, d, nranks, mode):
    from paper_2605_31425_b200 import shard
    C, R = workloads.config(k, m, d)
    dC = torch.from_numpy(C).cuda()
    dR = None if R is None else torch.from_numpy(R).cuda()
    pm = meb.MEB_MODE_FP64 if mode == "fp64" else meb.MEB_MODE_MIXED
    res = shard.ThreadRanks(nranks).solve(dC, dR, 1e-8, pm)
    co, ro, _ = ripalm.meb_solve(C, R, 1e-10, "fp64", ripalm.Params(dense_d_max=4096))
    c0, r0, st0 = res[0]
    for c, r, st in res:
        assert st["converged"] == 1
        assert r == r0 and torch.equal(c, c0)                       # bit-identical on every rank
    assert abs(r0 - ro) <= 1e-8 * ro and np.linalg.norm(c0.numpy() - co) <= 1e-5 * (1 + ro)
    assert _violation(C, R, c0.numpy(), r0) <= 1e-10 * (1 + r0)
    if mode == "mixed":
        assert sum(st["n_reduced"] for _, _, st in res) >= 1


def test_one_rank_sharded_equals_plain_solve(meb):
    """nranks = 1: same kernels, same initial point; only the order in which the per-CTA partials are added differs
    (packed sequentially into the record instead of lane-strided in the finalize kernel), so the two solves agree
    to rounding, not to the bit."""
    from paper_2605_31425_b200 import shard
    C, R = workloads.config(1, 8_000, 10)
    dC, dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
    (c1, r1, s1), = shard.ThreadRanks(1).solve(dC, dR, 1e-8, meb.MEB_MODE_MIXED)
    with meb.Context(*C.shape) as ctx:
        meb.meb_set_option(ctx, meb.OPT["NO_SMALL"], True)          # the sharded driver never uses the single-CTA solver
        c0, r0, s0 = meb.meb_solve(ctx, dC, dR, 1e-8, meb.MEB_MODE_MIXED)
    assert abs(r1 - r0) <= 1e-11 * r0 and np.linalg.norm(c1.numpy() - c0.numpy()) <= 1e-7 * (1 + r0)
    assert s1["converged"] == 1 and s0["converged"] == 1
