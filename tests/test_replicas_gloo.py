"""N > 1 path on CPU: world_size 2 over gloo (DESIGN.md §8 "replicas only").  Each rank builds its own pool
directory (host logic only, no device memory is touched), links its slice of the request list with
comb_link_plan, and rank 0 checks that the gathered per-rank tables are exactly the unsharded tables; the
max-over-ranks timing reduction bench.py relies on is checked in the same processes."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

import comb_synth as cs
from test_abi_host import make_pool, plan


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _tables(w, lo, hi):
    import paper_2602_01519_b200 as comb
    pool = make_pool(num_pages=w.pool_pages, Hkv=w.num_kv_heads, Dqk=w.head_dim_qk, Dv=w.head_dim_v, seed=11)
    for c in range(w.num_chunks):  # every replica stores the same population in the same order
        comb.comb_chunk_alloc(pool, c, int(w.chunk_len[c]))
    _, t = plan(pool, [list(map(int, w.links[r])) for r in range(lo, hi)])
    comb.comb_pool_destroy(pool)
    return t


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2602_01519_b200.replicas import max_over_ranks, shard_range
        w = cs.long_fewshot(requests=5, n_chunks=12, lq=4)  # ragged chunk lengths, odd request count
        lo, hi = shard_range(w.num_requests, rank, world)
        mine = _tables(w, lo, hi)
        gathered = [None] * world
        dist.all_gather_object(gathered, (lo, hi, mine))
        slowest = max_over_ranks(10.0 + rank)
        if rank == 0:
            full = _tables(w, 0, w.num_requests)
            assert [g[:2] for g in gathered] == [(0, 3), (3, 5)]
            ids = np.concatenate([g[2]["page_ids"] for g in gathered])
            ntok = np.concatenate([g[2]["page_ntok"] for g in gathered])
            kv = np.concatenate([g[2]["kv_len"] for g in gathered])
            tiles = np.concatenate([g[2]["tile_ntok"] for g in gathered])
            assert np.array_equal(ids, full["page_ids"]) and np.array_equal(ntok, full["page_ntok"])
            assert np.array_equal(kv, full["kv_len"]) and np.array_equal(tiles, full["tile_ntok"])
            off = 0
            for g in gathered:  # indptr of a shard = the unsharded indptr re-based at the shard's first request
                lo_g, hi_g, t = g
                assert np.array_equal(t["page_indptr"] + off, full["page_indptr"][lo_g:hi_g + 1])
                off += int(t["page_indptr"][-1])
            assert slowest == 10.0 + world - 1
        q.put((rank, "ok"))
    except Exception as e:  # surface the failure in the parent
        q.put((rank, repr(e)))
    finally:
        dist.destroy_process_group()


def test_two_replicas_shard_requests_and_reduce_max():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(30)
    assert res == {0: "ok", 1: "ok"}, res


def test_shard_range_partitions():
    from paper_2602_01519_b200.replicas import shard_range
    for n in (0, 1, 7, 128):
        for world in (1, 2, 3, 8):
            cuts = [shard_range(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
