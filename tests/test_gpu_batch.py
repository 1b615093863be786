"""GPU tests of meb_solve_batch (run with -m gpu): many small independent MEB instances, one CTA each.

Bar, per instance: radius within 1e-8 relative of the CPU oracle run to 1e-10, feasibility violation
<= 1e-10 (1 + r), the same answer (to 1e-9) as meb_solve on that instance alone."""
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


def _instances(specs, seed=0):
    Cs, Rs, offs = [], [], [0]
    any_r = any(has_r for _, _, has_r, _ in specs)
    for i, (m, d, has_r, kind) in enumerate(specs):
        rng = np.random.default_rng([seed, 77, i])
        if kind == "paper":
            C, R = workloads.paper_instance(m, d)
        elif kind == "sphere":
            g = rng.standard_normal((m, d)); C = g / np.linalg.norm(g, axis=1, keepdims=True); R = None
        else:
            C = rng.standard_normal((m, d)) * (1.0 + i); R = rng.uniform(0, 0.3, m) if has_r else None
        if any_r and R is None:
            R = np.zeros(m)
        Cs.append(np.ascontiguousarray(C, dtype=np.float64)); Rs.append(R); offs.append(offs[-1] + m)
    C = np.concatenate(Cs, 0)
    R = np.concatenate(Rs, 0) if any_r else None
    return C, R, np.array(offs, dtype=np.int64), Cs, Rs


def _violation(C, R, c, r):
    return float(np.max(np.sqrt(((C - c) ** 2).sum(1)) + (0 if R is None else R) - r))


def test_batch_matches_oracle_and_single_solves(meb):
    d = 20
    specs = [(1000, d, True, "gauss"), (37, d, True, "gauss"), (1, d, True, "gauss"), (4096, d, True, "gauss"),
             (500, d, False, "sphere"), (1000, d, True, "paper"), (333, d, True, "gauss"), (2, d, True, "gauss")]
    C, R, offs, Cs, Rs = _instances(specs)
    with meb.Context(int(offs[-1]), d) as ctx:
        dC = torch.from_numpy(C).cuda(); dR = torch.from_numpy(R).cuda()
        cb, rb, sb, kb = meb.meb_solve_batch(ctx, dC, dR, offs)
        assert (sb.numpy() == 0).all(), sb
        for k, (Ck, Rk) in enumerate(zip(Cs, Rs)):
            co, ro, _ = ripalm.meb_solve(Ck, Rk, 1e-10, "fp64")
            c, r = cb[k].numpy(), float(rb[k])
            assert abs(r - ro) <= 1e-8 * max(ro, 1e-300), (k, r, ro)
            assert np.linalg.norm(c - co) <= 1e-5 * (1 + ro)
            assert _violation(Ck, Rk, c, r) <= 1e-10 * (1 + r)
            assert float(kb[k]) <= 1e-8
            c1, r1, _ = meb.meb_solve(ctx, dC[offs[k]:offs[k + 1]], dR[offs[k]:offs[k + 1]], 1e-8, meb.MEB_MODE_FP64)
            assert abs(r1 - r) <= 1e-9 * (1 + r)


def test_batch_points_no_radii_and_wide_rows(meb):
    d = 126
    specs = [(300, d, False, "gauss"), (64, d, False, "gauss"), (1500, d, False, "gauss")]
    C, R, offs, Cs, Rs = _instances(specs, seed=3)
    assert R is None
    ld = d + 2                                            # padded rows
    Cp = np.zeros((C.shape[0], ld)); Cp[:, :d] = C
    with meb.Context(int(offs[-1]), d) as ctx:
        dC = torch.from_numpy(Cp).cuda()[:, :d]
        cb, rb, sb, kb = meb.meb_solve_batch(ctx, dC, None, offs)
        assert (sb.numpy() == 0).all()
        for k, Ck in enumerate(Cs):
            co, ro, _ = ripalm.meb_solve(Ck, None, 1e-10, "fp64")
            assert abs(float(rb[k]) - ro) <= 1e-8 * ro
            assert _violation(Ck, None, cb[k].numpy(), float(rb[k])) <= 1e-10 * (1 + ro)


def test_batch_degenerate_and_bad_instances(meb):
    d = 5
    rng = np.random.default_rng(5)
    good = rng.standard_normal((50, d))
    same = np.tile(rng.standard_normal(d), (7, 1))        # all balls are one point: r = 0
    bad = rng.standard_normal((9, d)); bad[4, 2] = np.nan
    C = np.concatenate([good, same, bad, good * 2], 0)
    R = np.zeros(C.shape[0])
    offs = np.array([0, 50, 57, 66, 116], dtype=np.int64)
    with meb.Context(int(offs[-1]), d) as ctx:
        cb, rb, sb, kb = meb.meb_solve_batch(ctx, torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda(), offs)
    s = sb.numpy()
    assert s[0] == 0 and s[1] == 0 and s[2] == meb.MEB_E_INPUT and s[3] == 0
    assert float(rb[1]) <= 1e-15 * np.abs(same[0]).max() and np.allclose(cb[1].numpy(), same[0], rtol=1e-15)
    co, ro, _ = ripalm.meb_solve(good, None, 1e-10, "fp64")
    assert abs(float(rb[0]) - ro) <= 1e-8 * ro and abs(float(rb[3]) - 2 * ro) <= 2e-8 * ro


def test_batch_rejects_oversized_instances(meb):
    with meb.Context(10000, 8) as ctx:
        dC = torch.zeros((5000, 8), dtype=torch.float64, device="cuda")
        with pytest.raises(meb.MebError) as ei:
            meb.meb_solve_batch(ctx, dC, None, np.array([0, 5000], dtype=np.int64))
        assert ei.value.code == meb.MEB_E_CAPACITY


def test_batch_is_deterministic_and_faster_than_a_loop(meb):
    d, m, nprob = 30, 1000, 296
    rng = np.random.default_rng(11)
    C = rng.standard_normal((m * nprob, d)) * rng.uniform(0.5, 2.0, (m * nprob, 1))
    offs = np.arange(nprob + 1, dtype=np.int64) * m
    with meb.Context(m * nprob, d) as ctx:
        dC = torch.from_numpy(C).cuda()
        a = meb.meb_solve_batch(ctx, dC, None, offs)
        b = meb.meb_solve_batch(ctx, dC, None, offs)
        assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
        assert (a[2].numpy() == 0).all()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record(); meb.meb_solve_batch(ctx, dC, None, offs); ev[1].record()
        for k in range(16):
            meb.meb_solve(ctx, dC[offs[k]:offs[k + 1]], None, 1e-8, meb.MEB_MODE_FP64)
        ev[2].record(); torch.cuda.synchronize()
        t_batch = ev[0].elapsed_time(ev[1]) / nprob
        t_loop = ev[1].elapsed_time(ev[2]) / 16
        print(f"batch: {t_batch * 1e3:.1f} us per instance; one at a time: {t_loop * 1e3:.1f} us per instance")
        assert t_batch < t_loop
