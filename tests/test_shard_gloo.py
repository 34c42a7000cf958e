"""world_size-2 gloo test (CPU) of the multi-GPU plumbing: batch shards, the F_q moment merge and the
max-over-ranks timing reduce.  The per-shard numbers come from the oracle, so the merged result
must equal the oracle's F_q of the whole batch."""
import dataclasses
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle as O
from paper_2606_22984_b200 import shard
from paper_2606_22984_b200 import workloads as W


def test_shard_bounds_cover_and_balance():
    for total in (1, 7, 1024, 4097):
        for world in (1, 2, 3, 8):
            b = [shard.shard_bounds(total, world, r) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == total
            assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = dataclasses.replace(W.CONFIGS["cfg2"], L=6, n_sites=36, window=5, n_layers=2)
    B = 37
    inp = W.make_all(w, batch=B)
    lo, hi = shard.shard_bounds(B, world, rank)
    u = inp["uniforms"][lo:hi]
    spins, lq, _ = O.sample(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"], u)
    E = O.energy_csr(spins, inp["bond_rowptr"], inp["bond_col"], inp["bond_val"])
    m_r, s_r = O.free_energy(E, lq, 0.7)          # the shard's own reduction (the GPU run takes fv_free_energy's)
    stats = torch.tensor([m_r, s_r, float(len(E)), s_r * s_r * len(E)], dtype=torch.float64)
    mean, std = shard.merge_free_energy(stats)
    tmax = shard.max_over_ranks(float(rank + 1))
    q.put((rank, lo, hi, mean, std, tmax))
    dist.destroy_process_group()


def test_two_rank_merge_matches_single_process():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = dataclasses.replace(W.CONFIGS["cfg2"], L=6, n_sites=36, window=5, n_layers=2)
    inp = W.make_all(w, batch=37)
    spins, lq, _ = O.sample(w, inp["weights"], inp["posemb"], inp["mask_rowptr"], inp["mask_col"], inp["uniforms"])
    E = O.energy_csr(spins, inp["bond_rowptr"], inp["bond_col"], inp["bond_val"])
    mean, std = O.free_energy(E, lq, 0.7)
    assert res[0][1:3] == (0, 19) and res[1][1:3] == (19, 37)
    for r in res:
        assert abs(r[3] - mean) < 1e-10 * abs(mean) and abs(r[4] - std) < 1e-8 * std
        assert r[5] == 2.0
