"""World-size-2 test of the sharded path's host logic on CPU (gloo): the partition, the rank-ordered all-gather
of per-rank records and the globalisation of index lists are the product's (paper_2605_31425_b200/shard.py); the
per-shard partials come from the ORACLE, and their rank-ordered combination must equal the oracle's evaluation of
the whole instance ("all-gather partials and sum in rank order")."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import primitives as prim
from paper_2605_31425_b200 import shard
from tests._gpu_common import make_state


def test_partition_is_contiguous_and_balanced():
    for m, n in [(10, 3), (7, 7), (1000003, 8), (5, 2), (2, 2)]:
        parts = shard.partition(m, n)
        assert parts[0][0] == 0 and sum(ml for _, ml in parts) == m
        for (o0, l0), (o1, l1) in zip(parts, parts[1:]):
            assert o0 + l0 == o1
        sizes = [ml for _, ml in parts]
        assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m, d = 1501, 12
        C, R, U, V, x, xbar = make_state(77, m, d)
        sigma, tau = 2.5, 0.7
        off, ml = shard.partition(m, world)[rank]
        sl = slice(off, off + ml)
        ev = prim.eval_alm(C[sl], R[sl], U[sl], V[sl], x, xbar, sigma, tau)
        # this rank's record: sums, maxima, counts, vector part (what csrc/meb_shard.cu packs)
        rec = np.concatenate([[ev["sum_proj2"], ev["sum_uplus"], ev["sum_dmult2"], ev["n_b1"], ev["n_b3"],
                               ev["max_pfeas"], ev["max_compl"], ev["max_dfeas"]], ev["sum_vplus"]])
        recs = shard.gather_records(torch.from_numpy(rec)).numpy()           # (world, 8 + d), rank order
        assert recs.shape == (world, 8 + d) and np.array_equal(recs[rank], rec)
        tot = recs[0].copy()
        for r in range(1, world):                                            # rank order
            tot[:5] += recs[r][:5]
            tot[5:8] = np.maximum(tot[5:8], recs[r][5:8])
            tot[8:] += recs[r][8:]
        full = prim.eval_alm(C, R, U, V, x, xbar, sigma, tau)
        assert abs(tot[0] - full["sum_proj2"]) <= 1e-13 * full["scale_proj2"]
        assert abs(tot[1] - full["sum_uplus"]) <= 1e-13 * full["scale_uplus"]
        assert abs(tot[2] - full["sum_dmult2"]) <= 1e-13 * full["scale_dmult2"]
        assert int(tot[3]) == full["n_b1"] and int(tot[4]) == full["n_b3"]
        assert tot[5] == full["max_pfeas"] and tot[6] == full["max_compl"]
        assert np.linalg.norm(tot[8:] - full["sum_vplus"]) <= 1e-13 * np.linalg.norm(full["scale_vplus"])
        # screening: local flags -> local compaction -> global indices; the sets concatenate in rank order
        C32 = C.astype(np.float32); R32 = R.astype(np.float32)
        tol_red = 0.4 * x[0]
        fl, _ = prim.screen_flags(C32[sl], R32[sl], x[0], x[1:], tol_red)
        loc = shard.globalize(torch.from_numpy(prim.compact(fl)), off)
        cnt = shard.gather_records(torch.tensor([loc.numel()], dtype=torch.int64)).view(-1)
        pad = torch.full((m,), -1, dtype=torch.int64)
        pad[:loc.numel()] = loc
        allidx = shard.gather_records(pad)
        cat = torch.cat([allidx[r, :int(cnt[r])] for r in range(world)]).numpy()
        ffull, _ = prim.screen_flags(C32, R32, x[0], x[1:], tol_red)
        assert np.array_equal(cat, np.flatnonzero(ffull)) and 0 < cat.size < m
        # feasibility: (delta_max, global argmax, violators) per rank -> max, smallest index on ties, sum
        dm, am, vi, _ = prim.feasibility_check(C[sl], R[sl], x[0], x[1:], 0.05)
        fr = shard.gather_records(torch.tensor([dm, float(am + off), float(vi.size)], dtype=torch.float64)).numpy()
        best = max(range(world), key=lambda r: (fr[r, 0], -fr[r, 1]))
        dmf, amf, vif, _ = prim.feasibility_check(C, R, x[0], x[1:], 0.05)
        assert fr[best, 0] == dmf and int(fr[best, 1]) == amf and int(fr[:, 2].sum()) == vif.size
        open(os.path.join(out_dir, f"ok{rank}"), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_rank_ordered_partials_equal_full_evaluation_world2(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all(os.path.exists(tmp_path / f"ok{r}") for r in range(world))
