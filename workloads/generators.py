"""Seeded generators for the five BASELINE.json configurations and the paper's LCG instances.

No arithmetic of the method lives here (no projections, no distances to a candidate
centre, no solver): only the random draws that define the input balls.

Recipe for ``config``: rows are generated in blocks of ``BLOCK_ROWS``
rows; block ``b`` of configuration ``k`` uses ``numpy.random.default_rng([seed, k, b])``
and draws that block's centres (row-major) first and then its radii.  Because the blocks
are independent, ``config(k, m=m')`` for ``m' < m`` is the first ``m'`` balls of the
full-size instance (except configuration 4, whose sphere/interior assignment is a
permutation of all ``m`` indices).
"""
from __future__ import annotations

import numpy as np

BLOCK_ROWS = 65536

# (m, d, has_radii) of BASELINE.json "configs"[0..4]  ->  k = 1..5
CONFIG_SHAPES = {
    1: (10_000, 10, True),
    2: (1_000_000, 100, False),
    3: (100_000, 1_000, True),
    4: (10_000_000, 32, False),
    5: (200_000, 10_000, True),
}


def _block(k: int, b: int, rows: int, d: int, seed: int, type_sphere=None):
    """Centres (rows x d) and radii (rows,) or None of block ``b`` of configuration ``k``."""
    rng = np.random.default_rng([seed, k, b])
    if k == 1:  # balls: centres N(0,1), radii U[0,0.1]
        C = rng.standard_normal((rows, d))
        R = rng.uniform(0.0, 0.1, rows)
    elif k == 2:  # points: centres N(0,1)
        C = rng.standard_normal((rows, d))
        R = None
    elif k == 3:  # balls: centres U[-1,1]^d, radii U[0,1]
        C = rng.uniform(-1.0, 1.0, (rows, d))
        R = rng.uniform(0.0, 1.0, rows)
    elif k == 4:  # boundary-heavy points: half on the unit sphere, half in the 0.99-ball
        G = rng.standard_normal((rows, d))
        G /= np.sqrt(np.sum(G * G, axis=1))[:, None]
        Uu = rng.uniform(0.0, 1.0, rows)
        scale = np.where(type_sphere, 1.0, 0.99 * Uu ** (1.0 / d))
        C = G * scale[:, None]
        R = None
    elif k == 5:  # anisotropic balls: centres N(0, diag(1/j)), radii log-normal(-3, 1)
        C = rng.standard_normal((rows, d))
        C *= (1.0 / np.sqrt(np.arange(1, d + 1, dtype=np.float64)))[None, :]
        R = rng.lognormal(mean=-3.0, sigma=1.0, size=rows)
    else:
        raise ValueError(f"unknown configuration {k}")
    return C, R


def config_blocks(k: int, m: int | None = None, d: int | None = None, seed: int = 0):
    """Yield ``(row0, C_block, R_block_or_None)`` block by block (streaming-friendly)."""
    m_full, d_full, _ = CONFIG_SHAPES[k]
    m = m_full if m is None else int(m)
    d = d_full if d is None else int(d)
    type_sphere_all = None
    if k == 4:
        perm = np.random.default_rng([seed, 4, 2**31 - 1]).permutation(m)
        type_sphere_all = perm < (m // 2)
    b = 0
    row0 = 0
    while row0 < m:
        rows = min(BLOCK_ROWS, m - row0)
        ts = None if type_sphere_all is None else type_sphere_all[row0:row0 + rows]
        # the block is always drawn at full BLOCK_ROWS length so that a prefix is a prefix
        Cb, Rb = _block(k, b, BLOCK_ROWS if k != 4 else rows, d, seed, ts)
        yield row0, Cb[:rows], (None if Rb is None else Rb[:rows])
        row0 += rows
        b += 1


def config(k: int, m: int | None = None, d: int | None = None, seed: int = 0):
    """Return ``(C, R)``: centres ``(m, d)`` float64 C-contiguous, radii ``(m,)`` float64 or None."""
    m_full, d_full, has_r = CONFIG_SHAPES[k]
    m = m_full if m is None else int(m)
    d = d_full if d is None else int(d)
    C = np.empty((m, d), dtype=np.float64)
    R = np.empty(m, dtype=np.float64) if has_r else None
    for row0, Cb, Rb in config_blocks(k, m, d, seed):
        C[row0:row0 + Cb.shape[0]] = Cb
        if R is not None:
            R[row0:row0 + Cb.shape[0]] = Rb
    return C, R


def config_into(k: int, C_out, R_out, m: int | None = None, d: int | None = None, seed: int = 0,
                threads: int = 8, sink=None):
    """Same rows as ``config`` written into preallocated ``C_out`` (m, d) / ``R_out`` (m,) (or handed block by
    block to ``sink(row0, C_block, R_block)``), the independent 65,536-row blocks drawn by a pool of threads
    (numpy's generators release the GIL).  Config 5 is 16 GB: one thread needs about a minute for it."""
    from concurrent.futures import ThreadPoolExecutor
    m_full, d_full, _ = CONFIG_SHAPES[k]
    m = m_full if m is None else int(m)
    d = d_full if d is None else int(d)
    type_sphere_all = None
    if k == 4:
        perm = np.random.default_rng([seed, 4, 2**31 - 1]).permutation(m)
        type_sphere_all = perm < (m // 2)
    nblocks = (m + BLOCK_ROWS - 1) // BLOCK_ROWS

    def work(b):
        row0 = b * BLOCK_ROWS
        rows = min(BLOCK_ROWS, m - row0)
        ts = None if type_sphere_all is None else type_sphere_all[row0:row0 + rows]
        Cb, Rb = _block(k, b, BLOCK_ROWS if k != 4 else rows, d, seed, ts)
        if sink is not None:
            sink(row0, Cb[:rows], None if Rb is None else Rb[:rows])
        else:
            C_out[row0:row0 + rows] = Cb[:rows]
            if R_out is not None and Rb is not None:
                R_out[row0:row0 + rows] = Rb[:rows]
        return rows

    with ThreadPoolExecutor(max_workers=max(1, int(threads))) as ex:
        return sum(ex.map(work, range(nblocks)))


def paper_instance(m: int, d: int):
    """The deterministic instances of the paper's experiments.

    psi_0 = 7, psi_{j+1} = (445 psi_j + 1) mod 4096, psibar_j = psi_j / 40.96 for j >= 1,
    assigned in the order r_1, c_1(1..d), r_2, c_2(1..d), ...
    """
    n = m * (d + 1)
    # the sequence has period 4096 (full-period LCG modulo 2^12): generate one period
    period = np.empty(4096, dtype=np.int64)
    psi = 7
    for j in range(4096):
        psi = (445 * psi + 1) % 4096
        period[j] = psi  # period[j] = psi_{j+1}
    seq = period[np.arange(n, dtype=np.int64) % 4096].astype(np.float64) / 40.96
    A = seq.reshape(m, d + 1)
    R = np.ascontiguousarray(A[:, 0])
    C = np.ascontiguousarray(A[:, 1:])
    return C, R
