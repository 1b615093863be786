"""The allocation-free entry point (include/meb.h a8', csrc/meb_static.cu) against the existing feasibility path.

Collected last on purpose (file name): the suite runs with ``pytest -x``.  The checks hold when this file runs alone in
a fresh process and when it runs after every other GPU test (the static scratch then still holds older contents).
"""
import numpy as np
import pytest
import torch

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200.binding as b
    b.load()
    return b


def _instance(seed, m, d, with_radii):
    rng = np.random.default_rng(seed)
    C = rng.standard_normal((m, d))
    R = rng.uniform(0.0, 0.3, size=m) if with_radii else None
    c = 0.1 * rng.standard_normal(d)
    r = 0.8 * float(np.sqrt(d))
    return C, R, c, r


def _compare(meb, ctx, Cd, Rd, cd, r, out):
    """One call of each path; returns (existing, static) results after the tolerance checks."""
    ref = meb.meb_feasibility_check(ctx, Cd, Rd, r, cd, 1e300)          # eps so large that no index list is written
    assert meb.meb_feasibility_max_static(Cd, Rd, r, cd, out) == meb.MEB_OK
    got = out.cpu().numpy()
    # the tolerance of tests/test_gpu_primitives.py::test_feasibility_check: 1e-12 of the magnitude of the terms
    dist = torch.sqrt(((Cd - cd) ** 2).sum(1))
    viol = dist + (Rd if Rd is not None else 0.0) - r
    scale = float((viol + r).abs().max()) + abs(r)
    assert abs(got[0] - ref["delta_max"]) <= 1e-12 * scale
    i = int(got[1])
    assert got[1] == i and 0 <= i < Cd.shape[0]
    assert float(viol[i]) >= ref["delta_max"] - 1e-12 * scale             # a maximiser (the order of rounding may differ)
    return ref, got


@pytest.mark.parametrize("m,d,with_radii,ld_pad", [(1, 1, False, 0), (257, 3, True, 5), (5000, 33, True, 0),
                                                   (70001, 100, False, 4), (3000, 1000, True, 0)])
def test_static_matches_existing_path_twice_in_a_row(meb, m, d, with_radii, ld_pad):
    out = torch.full((2,), -7.0, dtype=torch.float64, device="cuda")
    ctx = meb.Context(m, d)
    try:
        for call in range(2):                                            # two calls in a row share the scratch
            C, R, c, r = _instance(9000 + 13 * m + d + call, m, d, with_radii)
            if call == 1:                                                # fewer rows than the call before: stale tiles
                C, R = C[: max(1, m // 3)], (None if R is None else R[: max(1, m // 3)])
            buf = torch.zeros((C.shape[0], d + ld_pad), dtype=torch.float64, device="cuda")
            buf[:, :d] = torch.from_numpy(C).cuda()
            Cd = buf[:, :d]
            Rd = None if R is None else torch.from_numpy(R).cuda()
            cd = torch.from_numpy(c).cuda()
            _compare(meb, ctx, Cd, Rd, cd, r, out)
            again = out.clone()
            assert meb.meb_feasibility_max_static(Cd, Rd, r, cd, out) == meb.MEB_OK
            assert torch.equal(out, again)                               # deterministic, whatever the scratch held
    finally:
        ctx.close()


def test_static_argmax_tie_takes_smallest_index(meb):
    C = np.zeros((700, 4)); C[650] = [0, 0, -2, 0]; C[17] = [2, 0, 0, 0]; C[300] = [0, 2, 0, 0]
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    assert meb.meb_feasibility_max_static(torch.from_numpy(C).cuda(), None, 1.0, torch.zeros(4, dtype=torch.float64, device="cuda"),
                                          out) == meb.MEB_OK
    assert out.cpu().tolist() == [1.0, 17.0]


def test_static_on_paper_workload_and_side_stream(meb):
    """Config 2's shape (P:L394 of SURVEY: points N(0,1), d = 100) at a size of several waves, on a side stream."""
    m, d = 400_000, 100
    C, R = workloads.config(2, m=m, d=d, seed=3)[:2]
    Cd = torch.from_numpy(np.ascontiguousarray(C)).cuda()
    cd = torch.zeros(d, dtype=torch.float64, device="cuda")
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    ctx = meb.Context(m, d)
    try:
        s = torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            assert meb.meb_feasibility_max_static(Cd, None, 10.0, cd, out, stream=s) == meb.MEB_OK
        s.synchronize()
        first = out.clone()
        _compare(meb, ctx, Cd, None, cd, 10.0, out)
        assert torch.equal(first, out)
    finally:
        ctx.close()


def test_static_rejects_what_it_cannot_hold(meb):
    lib = meb.load()
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    p = x.data_ptr()
    too_many = meb.MEB_STATIC_MAX_ROWS + 1                               # no memory is touched: the size check comes first
    assert lib.meb_feasibility_max_static(None, too_many, 1, p, 1, None, 0.0, p, p) == meb.MEB_E_CAPACITY
    assert lib.meb_feasibility_max_static(None, 0, 1, p, 1, None, 0.0, p, p) == meb.MEB_E_ARG
    assert lib.meb_feasibility_max_static(None, 4, 2, p, 1, None, 0.0, p, p) == meb.MEB_E_ARG     # ld < d
    assert lib.meb_feasibility_max_static(None, 4, 2, None, 2, None, 0.0, p, p) == meb.MEB_E_ARG
