"""Pins for oracle/soc.py (CPU only).

The oracle's cone projection is pinned to things other than itself:
  * hand-evaluated examples of the printed formula P:L113-115 (tests/golden/),
  * the Moreau / KKT characterisation of a projection onto a self-dual cone:
    p = Pi_Q(z)  <=>  p in Q,  p - z in Q,  <p, p - z> = 0   (unique),
  * idempotence and the decomposition z = Pi_Q(z) - Pi_Q(-z),
  * the distance closed form (DESIGN reading 7),
  * central finite differences of the projection for the Clarke Jacobian element
    (DESIGN reading 1; the paper does not print P_i).
"""
import os

import numpy as np
import pytest

from oracle import soc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _examples():
    rows = []
    with open(os.path.join(GOLDEN, "soc_projection_examples.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            a, b, t, p = [s.split() for s in line.split("|")]
            rows.append((float(a[0]), [float(v) for v in b], float(t[0]), [float(v) for v in p]))
    return rows


def test_projection_hand_examples():
    ex = _examples()
    a = np.array([e[0] for e in ex])
    B = np.array([e[1] for e in ex])
    t, PV, br, nb = soc.proj_soc(a, B)
    np.testing.assert_allclose(t, [e[2] for e in ex], rtol=0, atol=1e-15)
    np.testing.assert_allclose(PV, [e[3] for e in ex], rtol=0, atol=1e-15)
    # branch of the examples, read off the printed conditions
    assert list(br) == [1, 1, 2, 2, 3, 3, 3, 3, 1, 2, 1]


def _rand_points(rng, m, d):
    a = rng.standard_normal(m) * 2
    B = rng.standard_normal((m, d))
    # put a third of the points exactly inside / in the polar cone
    B[: m // 3] *= 0.2
    return a, B


@pytest.mark.parametrize("d", [1, 2, 7, 33])
def test_projection_characterisation(d):
    rng = np.random.default_rng(100 + d)
    a, B = _rand_points(rng, 600, d)
    t, PV, br, nb = soc.proj_soc(a, B)
    assert set(np.unique(br)) == {1, 2, 3}
    scale = 1 + np.abs(a) + nb
    # p in Q
    assert np.all(np.sqrt((PV ** 2).sum(1)) <= t + 1e-14 * scale)
    # p - z in Q  (z - p in the polar cone -Q)
    assert np.all(np.sqrt(((PV - B) ** 2).sum(1)) <= (t - a) + 1e-14 * scale)
    # complementarity
    inner = t * (t - a) + np.sum(PV * (PV - B), axis=1)
    assert np.all(np.abs(inner) <= 1e-13 * scale ** 2)


def test_projection_idempotent_and_moreau():
    rng = np.random.default_rng(5)
    a, B = _rand_points(rng, 500, 6)
    t, PV, _, _ = soc.proj_soc(a, B)
    t2, PV2, _, _ = soc.proj_soc(t, PV)
    np.testing.assert_allclose(t2, t, atol=1e-14)
    np.testing.assert_allclose(PV2, PV, atol=1e-14)
    tm, PVm, _, _ = soc.proj_soc(-a, -B)       # Pi_Q(-z)
    np.testing.assert_allclose(t - tm, a, atol=1e-14)
    np.testing.assert_allclose(PV - PVm, B, atol=1e-14)


def test_dist_closed_form():
    # dist((a,b),Q) = 0 | sqrt(a^2+nb^2) | (nb - a)/sqrt(2)      (DESIGN reading 7)
    rng = np.random.default_rng(6)
    a, B = _rand_points(rng, 500, 5)
    nb = np.sqrt((B ** 2).sum(1))
    want = np.where(nb <= a, 0.0, np.where(nb <= -a, np.sqrt(a * a + nb * nb), (nb - a) / np.sqrt(2)))
    np.testing.assert_allclose(soc.dist_soc(a, B), want, atol=1e-14)
    # hand example: z = (0, (3,4)) -> projection (2.5, 1.5, 2) -> distance 5/sqrt(2)
    assert abs(soc.dist_soc(np.array([0.0]), np.array([[3.0, 4.0]]))[0] - 5 / np.sqrt(2)) < 1e-15


@pytest.mark.parametrize("d", [1, 3, 10])
def test_clarke_jacobian_finite_differences(d):
    rng = np.random.default_rng(7 + d)
    h = 1e-6
    n_b3 = 0
    for _ in range(60):
        a = float(rng.standard_normal()) * 1.5
        b = rng.standard_normal(d)
        nb = np.linalg.norm(b)
        if min(abs(nb - a), abs(nb + a)) < 1e-2:   # stay away from the branch boundaries
            continue
        P = soc.clarke_jacobian(a, b)
        z = np.concatenate([[a], b])
        J = np.empty((d + 1, d + 1))
        for j in range(d + 1):
            e = np.zeros(d + 1)
            e[j] = h
            tp, Pp, _, _ = soc.proj_soc(np.array([z[0] + e[0]]), (z[1:] + e[1:])[None, :])
            tm, Pm, _, _ = soc.proj_soc(np.array([z[0] - e[0]]), (z[1:] - e[1:])[None, :])
            J[:, j] = np.concatenate([tp - tm, (Pp - Pm)[0]]) / (2 * h)
        np.testing.assert_allclose(P, J, atol=2e-8)
        np.testing.assert_allclose(P, P.T, atol=0)
        assert np.linalg.eigvalsh(P).min() >= -1e-14        # PSD
        assert np.linalg.eigvalsh(P).max() <= 1 + 1e-14     # firmly nonexpansive
        n_b3 += int(abs(a) < nb)
    assert n_b3 >= 10
