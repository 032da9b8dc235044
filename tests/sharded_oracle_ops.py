"""CPU stand-in for the binding's four calls, backed by the oracle (test infrastructure): lets the
routing, reduction and merge of paper_2607_02525_b200/sharded.py run under gloo without a GPU."""
from types import SimpleNamespace

import numpy as np
import torch

import oracle


def _u64(t):
    return t.view(torch.int64).numpy().view(np.uint64)


class OracleOps:
    def __init__(self, radix_np=None):
        self.radix_np = radix_np

    def peek_block_hash(self, tokens, tok_off, nb):
        bo, h = oracle.block_hash(tokens.numpy(), tok_off.numpy(), 16, 0)
        return torch.from_numpy(bo), torch.from_numpy(h.view(np.int64)).view(torch.uint64)

    def peek_pending_tree(self, h, bo):
        t = oracle.pending_tree(_u64(h) if h.numel() else np.zeros(0, np.uint64), bo.numpy())
        return SimpleNamespace(order=torch.from_numpy(t.order), lcp=torch.from_numpy(t.lcp),
                               cluster_size=torch.from_numpy(t.cluster_size))

    def peek_lpm(self, tokens, tok_off, h, bo, radix=None, t_keys=None, tree=None):
        hr = hh = None
        if radix is not None:
            hr = torch.from_numpy(oracle.lpm_radix(tokens.numpy(), tok_off.numpy(), radix))
        if t_keys is not None:
            hh = torch.from_numpy(oracle.lpm_hash(_u64(h) if h.numel() else np.zeros(0, np.uint64), bo.numpy(), _u64(t_keys)))
        return hr, hh

    def peek_demand_rank(self, h, bo, tree=None, t_keys=None, hit=None, cluster_size=None, arrival=None,
                         want_demand=None, want_order=None):
        dem = order = None
        if want_demand:
            dem = torch.from_numpy(oracle.demand(_u64(h) if h.numel() else np.zeros(0, np.uint64), bo.numpy(), _u64(t_keys)))
        if want_order:
            order = torch.from_numpy(oracle.clpm_order(hit.numpy(), cluster_size.numpy(),
                                                        arrival.numpy() if arrival is not None else None))
        return dem, order
