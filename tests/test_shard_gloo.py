"""N > 1 path on CPU: two `gloo` ranks shard the templates.

The path has no exchange step, so what needs covering is the host logic: shards are
disjoint, whole banks, cover every template; a rank's sub-bank reproduces exactly its
rows of the full bank's output (templates are independent); merged
trigger lists carry global template indices; timing is the max over ranks.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import workloads
from paper_2011_06787_b200 import shard as shd
from paper_2011_06787_b200.binding import TRIGGER_DTYPE


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_template_shard_partitions_whole_banks():
    for n_t, world, bs in [(20000, 8, 1000), (4000, 3, 1000), (10, 4, 1), (7, 2, 4), (3, 5, 1)]:
        spans = [shd.template_shard(r, world, n_t, bs) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == n_t
        for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
            assert a1 == b0 and a0 <= a1
        for t0, t1 in spans:
            assert t0 % bs == 0 and (t1 % bs == 0 or t1 == n_t)
        n_banks = [-(-(t1 - t0) // bs) for t0, t1 in spans]
        assert max(n_banks) - min(n_banks) <= 1
    with pytest.raises(ValueError):
        shd.template_shard(2, 2, 10)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(5)
        bank = workloads.random_bank(rng, 6, 12, [2048], out_band=0)
        x = workloads.gaussian_strain(np.random.default_rng(6), 2, 1024)
        t0, t1 = shd.template_shard(rank, world, bank["n_templates"], bank_size=2)
        sub = shd.slice_bank(bank, t0, t1)
        z_sub = oracle.filter_bank(x, sub)
        z_full = oracle.filter_bank(x, bank)
        same = bool(np.array_equal(z_sub, z_full[:, t0:t1]))
        # local triggers: one per (det, local template), every second one valid
        D, T = 2, t1 - t0
        k, _ = oracle.peaks_mode0(np.ascontiguousarray(z_sub.astype(np.complex64)).reshape(D * T, -1), 0.0)
        loc = np.zeros(D * T, TRIGGER_DTYPE)
        loc["tmpl"] = np.tile(np.arange(T), D)
        loc["det"] = np.repeat(np.arange(D), T)
        loc["k"] = k
        loc["valid"] = (np.arange(D * T) % 2 == 0)
        merged = shd.merge_triggers(loc, t0)
        mx = shd.max_over_ranks(10.0 + rank)
        sm = shd.sum_over_ranks(float(T))
        q.put((rank, t0, t1, same, merged, mx, sm, int(loc["valid"].sum())))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_without_exchange():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted([q.get(timeout=180) for _ in range(world)], key=lambda o: o[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, a0, a1, same0, m0, mx0, sm0, nv0), (r1, b0, b1, same1, m1, mx1, sm1, nv1) = out
    assert (a0, a1, b0, b1) == (0, 4, 4, 6)               # 3 banks of 2: rank 0 takes the extra bank
    assert same0 and same1                                 # a shard is an exact sub-problem
    assert mx0 == mx1 == 11.0 and sm0 == sm1 == 6.0        # slowest rank sets the time; units add up
    assert len(m0) == len(m1) == nv0 + nv1                 # every rank sees every valid trigger
    assert np.array_equal(m0, m1)
    assert set(m0["tmpl"][:nv0]) <= set(range(0, 4)) and set(m0["tmpl"][nv0:]) <= set(range(4, 6))
    assert np.all(m0["valid"] == 1)
