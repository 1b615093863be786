"""Over-read guard ("What's missing" 7: compute-sanitizer is closed on this pool).

Every input array of a call -- C (with its row padding), R, U, the slot map, the V pool -- is placed so that
it ends exactly where a guard region begins; the guard and the row padding hold NaN (slot map: a huge index).
A kernel that reads past the end of a caller's buffer, or that lets padding values into its arithmetic
(bulk copies and 128-bit loads fetch whole 16-byte units), poisons its outputs with NaN or leaves the
allocation, and the results stop being bit-identical to the same call on plain zero-padded arrays."""
import numpy as np
import pytest
import torch

from tests._gpu_common import dvec, make_state

pytestmark = pytest.mark.gpu
THDT = {0: torch.float64, 1: torch.float32}
GUARD = 4096          # elements


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    meb.load()
    return meb


@pytest.fixture(scope="module")
def ctx(meb):
    c = meb.Context(1 << 15, 4096)
    yield c
    c.close()


def _guarded(t, fill):
    """A copy of the 1-D/2-D tensor `t` that ends flush against a guard region filled with `fill`."""
    flat = t.reshape(-1)
    n = flat.numel()
    buf = torch.full((n + GUARD,), fill, dtype=t.dtype, device=t.device)      # same (aligned) start as a plain allocation
    buf[:n].copy_(flat)
    return buf[:n].view(t.shape), buf


def _device_state(C, R, U, V, prec, ld_pad, guarded):
    dt = THDT[prec]
    dev = torch.device("cuda")
    m, d = C.shape
    ld = d + ld_pad
    nan = float("nan")
    Cfull = torch.full((m, ld), nan if guarded else 0.0, dtype=dt, device=dev)
    Cfull[:, :d] = torch.from_numpy(C).to(dt).to(dev)
    rows = np.flatnonzero(U > 0)
    ldv = (d + 3) // 4 * 4
    Vfull = torch.full((max(rows.size, 1), ldv), nan if guarded else 0.0, dtype=dt, device=dev)
    Vfull[:rows.size, :d] = torch.from_numpy(V[rows]).to(dt).to(dev)
    slot_h = np.full(m, -1, dtype=np.int32)
    slot_h[rows] = np.arange(rows.size, dtype=np.int32)
    Rt = torch.from_numpy(R).to(dt).to(dev)
    Ut = torch.from_numpy(U).to(dt).to(dev)
    St = torch.from_numpy(slot_h).to(dev)
    keep = []
    if guarded:
        Cfull, b0 = _guarded(Cfull, nan)
        Vfull, b1 = _guarded(Vfull, nan)
        Rt, b2 = _guarded(Rt, nan)
        Ut, b3 = _guarded(Ut, nan)
        St, b4 = _guarded(St, 0x7FFFFFF0)
        keep = [b0, b1, b2, b3, b4]
    return Cfull[:, :d], Rt, Ut, St, Vfull[:, :d], keep


SHAPES = [(1000, 10, 0), (1203, 5, 1), (999, 32, 0), (3001, 100, 0), (513, 257, 1), (257, 33, 0), (300, 1000, 0),
          (70, 2600, 0), (41, 2500, 0)]


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("m,d,ld_pad", SHAPES)
def test_no_over_read_and_padding_is_ignored(meb, ctx, prec, m, d, ld_pad):
    C, R, U, V, x, xbar = make_state(1300 + m + d, m, d)
    f = (lambda a: a.astype(np.float32).astype(np.float64)) if prec == 1 else (lambda a: a)
    C, R, U, V = f(C), f(R), f(U), f(V)
    outs = []
    for guarded in (False, True):
        Cd, Rd, Ud, Sd, Vd, keep = _device_state(C, R, U, V, prec, ld_pad, guarded)
        ev = meb.meb_eval_alm(ctx, prec, Cd, Rd, Ud, Sd, Vd, dvec(x), dvec(xbar), 2.0, 0.5, per_ball=True, active=True)
        q = dvec(np.random.default_rng(3).standard_normal(d + 1))
        Hq = meb.meb_hvp(ctx, prec, Cd, Rd, Ud, Sd, Vd, dvec(x), 2.0, 0.5, q)
        up = meb.meb_update_multipliers(ctx, prec, Cd, Rd, Ud, Sd, Vd, dvec(x), 1.7)
        res = [ev["scalars"], ev["grad"], ev["t"], ev["lam"], ev["active_idx"], ev["active_rho"], Hq,
               up["U"], up["v_slot"], up["Vrows"], torch.tensor([up["sum_mult2"]])]
        if prec == 0:
            fe = meb.meb_feasibility_check(ctx, Cd, Rd, float(x[0]), dvec(x[1:]), 0.05)
            ing = meb.meb_ingest(ctx, Cd, Rd, 1024, want_shadow=True)
            res += [torch.tensor([fe["delta_max"], float(fe["argmax"])]), fe["viol_idx"], ing["c0"],
                    torch.tensor([ing["L"], float(ing["n_bad"])]), ing["C32"], ing["R32"]]
            if d <= 128:
                res.append(meb.meb_dense_hessian(ctx, prec, Cd, Rd, Ud, Sd, Vd, dvec(x), 2.0, 0.5))
        else:
            sc = meb.meb_screen_compact(ctx, Cd, Rd, float(x[0]), dvec(x[1:]), 0.1 * float(x[0]))
            res += [sc["idx"], sc["flags"]]
        outs.append([r.detach().cpu().clone() for r in res])
        del keep
    for a, b in zip(*outs):
        assert not torch.isnan(b.double()).any()
        assert torch.equal(a, b)
