"""one queue sharded over G ranks by the first block's hash - world 2 on CPU
(gloo).  The per-shard compute is the oracle's (tests/sharded_oracle_ops.py); what is tested is the
path's own logic: ownership, sub-queues, the all-reduce of demand, the all-gather and merge of the
cLPM keys.  The merged result must equal the unsharded oracle result, every element."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _inputs(cfg, seed):
    import oracle
    from harness import workloads as W
    wl = W.make(cfg, seed=seed, small=True)
    toks, off = wl.queue.materialize_np()
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    return wl, toks, off, cache


def _orc_radix(r):
    import oracle
    return oracle.Radix(r.c_tokens, r.n_tok_off, r.n_tok_len, r.n_child_off, r.e_first_tok, r.e_child)


def _worker(rank, world, port, cfg, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2607_02525_b200 import sharded
    from sharded_oracle_ops import OracleOps
    wl, toks, off, cache = _inputs(cfg, 42)
    radix = _orc_radix(cache.radix) if cache.radix is not None else None
    keys = torch.from_numpy(cache.t_keys.view(np.int64)).view(torch.uint64)
    res = sharded.sharded_step(OracleOps(), torch.from_numpy(toks), torch.from_numpy(off),
                               torch.from_numpy(wl.arrival), radix, keys, int(keys.shape[0]), rank, world, dist)
    out[rank] = (res.hit.numpy(), res.cluster_size.numpy(), res.demand.numpy(), res.clpm_order.numpy(), res.owner.numpy())
    dist.barrier()
    dist.destroy_process_group()


def _check(cfg):
    import oracle
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), cfg, out), nprocs=world, join=True)
    wl, toks, off, cache = _inputs(cfg, 42)
    bo, h = oracle.block_hash(toks, off, 16, 0)
    tree = oracle.pending_tree(h, bo)
    hit = oracle.lpm_radix(toks, off, _orc_radix(cache.radix)) if cache.radix is not None else oracle.lpm_hash(h, bo, cache.t_keys)
    demand = oracle.demand(h, bo, cache.t_keys)
    order = oracle.clpm_order(hit, tree.cluster_size, wl.arrival)
    for r in range(world):
        g_hit, g_cs, g_dem, g_ord, owner = out[r]
        assert np.array_equal(g_hit, hit)
        assert np.array_equal(g_cs, tree.cluster_size)   # a cluster never spans two shards
        assert np.array_equal(g_dem, demand)             # sum over the shards = the queue's demand
        assert np.array_equal(g_ord, order)              # merged cLPM order, ties included
    owner = out[0][4]
    assert set(np.unique(owner).tolist()) <= {0, 1}
    # requests that share their first block have one owner
    nb = np.diff(bo)
    k0 = h[bo[:-1][nb > 0]]
    own = owner[nb > 0]
    for key in np.unique(k0)[:50]:
        assert len(set(own[k0 == key].tolist())) == 1


def test_sharded_queue_world2_config1():
    _check(1)


def test_sharded_queue_world2_config4_table_only():
    _check(4)
