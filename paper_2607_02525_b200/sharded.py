"""One queue sharded over G GPUs - an opt-in mode beside the default
"one independent PEEK instance per replica".

Requests whose chains start with different first blocks never share a node of the pending trie, so
the queue is partitioned by the chained hash of the first block, `k_0 mod G` (requests without a
full block go by index): every GPU's sub-forest is independent.  Routing happens at arrival - the
router hashes a prompt's first 16 tokens - so the data path has no all-to-all; the cache arrays are
replicated (read-only).  Per cycle every rank runs the four calls on its own requests; then
    demand      one all-reduce (sum) of int32[S]      - a slot's demand is a sum over requests
    cLPM order  one all-gather of (hit, cluster size, request) - 12 bytes per request - and the same
                sort as on one GPU over the gathered keys
Cluster and group signals need no exchange: a cluster never spans two shards.  Skew caveat: a queue
whose prompts all share block 0 (configs[2]) degenerates to one owner; shard such a workload by
replicas instead.

This module is argument routing around the library calls (`ops`) and `torch.distributed`
collectives; every step of the path still runs in the kernels behind `ops`.  `ops` is any object
with the binding's four functions (the tests pass a CPU stand-in so that the routing, the reduction
and the merge are covered with gloo on machines without a GPU).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import torch


@dataclass
class ShardResult:
    hit: torch.Tensor           # int32[N]  by global request index
    cluster_size: torch.Tensor  # int32[N]
    demand: torch.Tensor        # int32[S]  summed over the shards
    clpm_order: torch.Tensor    # int32[N]  global admission order
    owner: torch.Tensor         # int32[N]  rank that owns each request


def first_block_owner(ops, tokens: torch.Tensor, tok_off: torch.Tensor, G: int) -> torch.Tensor:
    """owner[r] = k^r_0 mod G (unsigned), r mod G for a request without a full block.  k_0 comes from
    `ops.peek_block_hash` over the first 16 tokens of every request (what a router computes at arrival)."""
    N = int(tok_off.shape[0]) - 1
    lens = tok_off[1:] - tok_off[:-1]
    has = lens >= 16
    take = torch.where(has, torch.full_like(lens, 16), torch.zeros_like(lens))
    off16 = torch.zeros(N + 1, dtype=torch.int64, device=tok_off.device)
    off16[1:] = torch.cumsum(take, 0)
    idx = (tok_off[:-1][has].unsqueeze(1) + torch.arange(16, device=tok_off.device).unsqueeze(0)).reshape(-1)
    first = tokens[idx].contiguous() if idx.numel() else tokens[:0].contiguous()
    nb = int(has.sum().item())
    _, k0 = ops.peek_block_hash(first, off16, nb)
    owner = torch.arange(N, dtype=torch.int64, device=tok_off.device) % G
    if nb:
        k = k0.view(torch.int64)[:nb]
        # unsigned k mod G from the signed view: ((k >> 1) mod G * 2 + (k & 1)) mod G
        m = (((k >> 1) & 0x7FFFFFFFFFFFFFFF) % G * 2 + (k & 1)) % G
        owner[has] = m
    return owner.to(torch.int32)


def sub_queue(tokens: torch.Tensor, tok_off: torch.Tensor, mine: torch.Tensor):
    """CSR of the requests `mine` (ascending global indices)."""
    lens = (tok_off[1:] - tok_off[:-1])[mine]
    off = torch.zeros(mine.numel() + 1, dtype=torch.int64, device=tok_off.device)
    off[1:] = torch.cumsum(lens, 0)
    T = int(off[-1].item())
    if T == 0:
        return tokens[:0].contiguous(), off
    starts = tok_off[:-1][mine]
    rep = torch.repeat_interleave(torch.arange(mine.numel(), device=tok_off.device), lens)
    pos = torch.arange(T, device=tok_off.device) - off[:-1][rep] + starts[rep]
    return tokens[pos].contiguous(), off


def local_pass(ops, tokens, tok_off, arrival, radix, t_keys, S: int):
    """The four calls on one shard's requests.  Returns (hit, cluster_size, demand)."""
    n = int(tok_off.shape[0]) - 1
    dev = tok_off.device
    if n == 0:
        return (torch.zeros(0, dtype=torch.int32, device=dev), torch.zeros(0, dtype=torch.int32, device=dev),
                torch.zeros(S, dtype=torch.int32, device=dev))
    nb = int(((tok_off[1:] - tok_off[:-1]) // 16).sum().item())
    bo, h = ops.peek_block_hash(tokens, tok_off, nb)
    tree = ops.peek_pending_tree(h, bo)
    hr, hh = ops.peek_lpm(tokens, tok_off, h, bo, radix=radix, t_keys=t_keys, tree=tree)
    hit = hr if hr is not None else hh
    if t_keys is not None:
        demand, _ = ops.peek_demand_rank(h, bo, tree=tree, t_keys=t_keys, hit=None, cluster_size=None, arrival=None,
                                         want_demand=True, want_order=False)
    else:
        demand = torch.zeros(S, dtype=torch.int32, device=dev)
    return hit, tree.cluster_size, demand


def merge(ops, N: int, parts, arrival: Optional[torch.Tensor]):
    """parts: per rank (global indices, hit, cluster_size).  Scatters them into request order and sorts
    the gathered cLPM keys with the library's own rank call: the single-GPU order, ties included."""
    dev = parts[0][0].device
    hit = torch.zeros(N, dtype=torch.int32, device=dev)
    cs = torch.zeros(N, dtype=torch.int32, device=dev)
    for gidx, h, c in parts:
        hit[gidx.long()] = h
        cs[gidx.long()] = c
    _, order = ops.peek_demand_rank(None, None, tree=None, t_keys=None, hit=hit, cluster_size=cs, arrival=arrival,
                                    want_demand=False, want_order=True)
    return hit, cs, order


def sharded_step(ops, tokens, tok_off, arrival, radix, t_keys, S: int, rank: int, G: int, dist=None) -> ShardResult:
    """One cycle on rank `rank` of G.  `dist` = torch.distributed (initialised) or None for G == 1.
    Every rank is given the queue as it arrived (tokens / tok_off replicated here; a router would hand
    each rank only its own requests) and returns the global result."""
    N = int(tok_off.shape[0]) - 1
    dev = tok_off.device
    owner = first_block_owner(ops, tokens, tok_off, G)
    mine = torch.nonzero(owner == rank).squeeze(1)
    tok_l, off_l = sub_queue(tokens, tok_off, mine)
    arr_l = arrival[mine].contiguous() if arrival is not None else None
    hit_l, cs_l, demand = local_pass(ops, tok_l, off_l, arr_l, radix, t_keys, S)
    if G == 1 or dist is None:
        parts = [(mine.to(torch.int32), hit_l, cs_l)]
    else:
        dist.all_reduce(demand, op=dist.ReduceOp.SUM)  # int32[S]: a slot's demand is a sum over requests
        counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(G)]
        dist.all_gather(counts, torch.tensor([mine.numel()], dtype=torch.int64, device=dev))
        cap = int(max(int(c.item()) for c in counts))
        pack = torch.zeros(3, max(cap, 1), dtype=torch.int32, device=dev)  # request, hit, cluster size: 12 bytes each
        pack[0, : mine.numel()] = mine.to(torch.int32)
        pack[1, : mine.numel()] = hit_l
        pack[2, : mine.numel()] = cs_l
        got = [torch.zeros_like(pack) for _ in range(G)]
        dist.all_gather(got, pack)
        parts = [(g[0, : int(c.item())], g[1, : int(c.item())], g[2, : int(c.item())]) for g, c in zip(got, counts)]
    hit, cs, order = merge(ops, N, parts, arrival)
    return ShardResult(hit, cs, demand, order, owner)


def sharded_step_emulated(ops, tokens, tok_off, arrival, radix, t_keys, S: int, G: int) -> ShardResult:
    """The same cycle with the G ranks run one after the other on ONE device (no kernel waits for
    another rank): the collectives become a sum and a concatenation.  Test and single-GPU use."""
    N = int(tok_off.shape[0]) - 1
    owner = first_block_owner(ops, tokens, tok_off, G)
    demand = None
    parts = []
    for rank in range(G):
        mine = torch.nonzero(owner == rank).squeeze(1)
        tok_l, off_l = sub_queue(tokens, tok_off, mine)
        arr_l = arrival[mine].contiguous() if arrival is not None else None
        hit_l, cs_l, d = local_pass(ops, tok_l, off_l, arr_l, radix, t_keys, S)
        demand = d if demand is None else demand + d
        parts.append((mine.to(torch.int32), hit_l, cs_l))
    hit, cs, order = merge(ops, N, parts, arrival)
    return ShardResult(hit, cs, demand, order, owner)
