"""peek_block_hash_static: the block hash with its scratch in a static device array inside the library
(include/peek.h), for callers that cannot allocate device memory.  Checked against the existing
path (peek_block_hash with a caller-provided workspace), bit-exact like every other parity test here
(integer work), on calls in a row that share the static array.

This file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide
the parity tests.  It passes alone in a fresh process and after the other tests."""
import ctypes

import numpy as np
import pytest
import torch

from harness import workloads as W

DEV = "cuda:0"


def _b():
    from paper_2607_02525_b200 import binding
    return binding


def _queue(cfg, seed):
    wl = W.make(cfg, seed=seed, small=True)
    toks, off = wl.queue.materialize_np()
    return toks, off, int((np.diff(off) // 16).sum())


def _ragged_queue(n, seed):
    """n requests of 0..300 tokens (empty ones, ragged tails, arbitrary start alignment)."""
    rng = np.random.default_rng(seed)
    lens = rng.integers(0, 301, size=n)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    toks = rng.integers(0, 128256, size=int(off[-1])).astype(np.int32)
    return toks, off, int((lens // 16).sum())


def test_static_rejects_sizes_beyond_the_maximum():
    """N above PEEK_BLOCK_HASH_STATIC_MAX_N answers PEEK_ERR_CAPACITY from the host-side checks, before
    any pointer is looked at or any CUDA call is made (so this runs without a GPU)."""
    b = _b()
    L = b.lib()
    dummy = (ctypes.c_int64 * 4)()
    p = ctypes.cast(dummy, ctypes.c_void_p)
    st = L.peek_block_hash_static(p, p, b.BLOCK_HASH_STATIC_MAX_N + 1, 16, ctypes.c_uint64(0), p, p, 0, None)
    assert st == -2  # PEEK_ERR_CAPACITY
    msg = L.peek_last_error().decode()
    assert "static scratch" in msg and str(b.BLOCK_HASH_STATIC_MAX_N) in msg
    assert L.peek_block_hash_static(p, p, -1, 16, ctypes.c_uint64(0), p, p, 0, None) == -1
    assert L.peek_block_hash_static(p, p, 0, 16, ctypes.c_uint64(0), p, p, 0, None) == 0  # N = 0 touches nothing


@pytest.mark.gpu
def test_static_matches_workspace_path_on_calls_in_a_row():
    b = _b()
    # a queue on the three-launch scan (N > 8192), then one on the one-launch scan, then the first
    # again: every call finds the previous call's partial sums and counter in the shared array
    cases = [_ragged_queue(20000, 11), _queue(1, 12), _queue(2, 13), _ragged_queue(20000, 11)]
    assert cases[0][1].shape[0] - 1 > 8192 and cases[1][1].shape[0] - 1 <= 8192
    free_before = None
    for i, (toks, off, NB) in enumerate(cases):
        d_tok = torch.from_numpy(toks).to(DEV)
        d_off = torch.from_numpy(off).to(DEV)
        N = off.shape[0] - 1
        ref_bo, ref_h = b.peek_block_hash(d_tok, d_off, NB, seed=7)
        bo = torch.full((N + 1,), -1, dtype=torch.int64, device=DEV)
        h = torch.zeros(max(NB, 1), dtype=torch.uint64, device=DEV)
        torch.cuda.synchronize()
        if i > 0:  # the first call may load the module lazily; from then on nothing may be allocated
            free_before = torch.cuda.mem_get_info()[0]
        for rep in range(2):  # two calls in a row on the same inputs
            g_bo, g_h = b.peek_block_hash_static(d_tok, d_off, NB, bo, h, seed=7)
            torch.cuda.synchronize()
            assert torch.equal(g_bo, ref_bo), "blk_off differs (case %d, call %d)" % (i, rep)
            assert torch.equal(g_h.view(torch.int64), ref_h.view(torch.int64)), "hashes differ (case %d, call %d)" % (i, rep)
            h.zero_()
            bo.fill_(-1)
        if free_before is not None:
            assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was allocated by the call"
