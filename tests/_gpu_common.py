"""Helpers shared by the GPU parity tests: seeded evaluation states (numpy only, no method
arithmetic beyond drawing multipliers inside Q) and conversion to the library's sparse V layout."""
import numpy as np
import torch


def make_state(seed, m, d, with_radii=True, frac_mult=0.3, data="normal"):
    """A generic, non-converged evaluation point: ~30% of the balls stick out of the current ball,
    a fraction of the balls carries multipliers (u_i, v_i) in Q."""
    rng = np.random.default_rng(seed)
    if data == "normal":
        C = rng.standard_normal((m, d))
    else:
        C = rng.uniform(-1, 1, (m, d))
    R = rng.uniform(0, 0.3, m) if with_radii else None
    c = rng.standard_normal(d) * 0.1
    dist = np.sqrt(((C - c) ** 2).sum(1)) + (0 if R is None else R)
    r = float(np.quantile(dist, 0.7)) * 1.0001   # off the data points: no ball exactly on a branch boundary
    x = np.concatenate([[r], c])
    xbar = x + rng.standard_normal(d + 1) * 0.05
    U = np.zeros(m)
    V = np.zeros((m, d))
    k = int(frac_mult * m)
    if k > 0:
        idx = np.sort(rng.permutation(m)[:k])
        U[idx] = rng.uniform(0.01, 1.0, k)
        dirs = rng.standard_normal((k, d))
        dirs /= np.sqrt((dirs ** 2).sum(1))[:, None]
        V[idx] = dirs * (U[idx] * rng.uniform(0, 1, k))[:, None]
        U[idx[: max(1, k // 20)]] += 30.0        # a few balls deep inside Q: branch B1
    return C, R, U, V, x, xbar


def to_device(C, R, U, V, prec_dtype, layout="sparse", ld_pad=0):
    """layout: 'none' (no multipliers), 'sparse' (rows with u_i > 0 only), 'dense' (slot[i] = i)."""
    dev = torch.device("cuda")
    m, d = C.shape
    ld = d + ld_pad
    Cd = torch.zeros((m, ld), dtype=prec_dtype, device=dev)
    Cd[:, :d] = torch.from_numpy(C).to(prec_dtype).to(dev)
    Cd = Cd[:, :d]
    Rd = None if R is None else torch.from_numpy(R).to(prec_dtype).to(dev)
    if layout == "none":
        return Cd, Rd, None, None, None
    Ud = torch.from_numpy(U).to(prec_dtype).to(dev)
    ldv = (d + 3) // 4 * 4
    if layout == "dense":
        slot = torch.arange(m, dtype=torch.int32, device=dev)
        Vr = torch.zeros((m, ldv), dtype=prec_dtype, device=dev)
        Vr[:, :d] = torch.from_numpy(V).to(prec_dtype).to(dev)
    else:
        rows = np.flatnonzero(U > 0)
        slot_h = np.full(m, -1, dtype=np.int32)
        perm = np.random.default_rng(1).permutation(rows.size)      # slots in scrambled order
        slot_h[rows] = perm.astype(np.int32)
        Vr = torch.zeros((max(rows.size, 1), ldv), dtype=prec_dtype, device=dev)
        Vh = np.zeros((max(rows.size, 1), d))
        Vh[perm] = V[rows]
        Vr[:, :d] = torch.from_numpy(Vh).to(prec_dtype).to(dev)
        slot = torch.from_numpy(slot_h).to(dev)
    return Cd, Rd, Ud, slot, Vr[:, :d]


def dvec(x):
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).cuda()
