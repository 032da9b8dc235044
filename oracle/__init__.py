"""CPU oracle for the PEEK hot path — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes loader around ``oracle/peek_oracle.cpp`` (plain C++17, see the header
of that file for what each function follows in the paper and how it is pinned).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  Nothing under
``paper_2607_02525_b200/`` imports it and it imports nothing from there.

All arrays are numpy, C-contiguous, with the dtypes of SURVEY.md section 8(a).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "peek_oracle.cpp")
_LIB = os.path.join(_HERE, "libpeek_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (building the checker is not using it)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", _SRC, "-o", _LIB]
    subprocess.run(cmd, check=True)
    return _LIB


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ct))


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.orc_mix64_export.restype = ctypes.c_uint64
        L.orc_mix64_export.argtypes = [ctypes.c_uint64]
        L.orc_position_multiplier.restype = ctypes.c_uint64
        L.orc_position_multiplier.argtypes = [ctypes.c_int32]
        L.orc_block_hash.restype = ctypes.c_int64
        L.orc_num_threads.restype = ctypes.c_int
        L.orc_has_sharing.restype = ctypes.c_int32
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(ctypes.c_int(int(n)))


def mix64(x: int) -> int:
    return int(lib().orc_mix64_export(ctypes.c_uint64(x & (2**64 - 1))))


def position_multiplier(j: int) -> int:
    return int(lib().orc_position_multiplier(ctypes.c_int32(j)))


def _c(a, dt):
    a = np.ascontiguousarray(a, dtype=dt)
    return a


I32, I64, U64 = ctypes.c_int32, ctypes.c_int64, ctypes.c_uint64


def block_hash(tokens, tok_off, block_size: int = 16, seed: int = 0):
    """O1.  Returns (blk_off int64[N+1], hashes uint64[NB])."""
    tokens = _c(tokens, np.int32)
    tok_off = _c(tok_off, np.int64)
    N = tok_off.shape[0] - 1
    blk_off = np.zeros(N + 1, dtype=np.int64)
    NB = lib().orc_block_hash(_p(tokens, I32), _p(tok_off, I64), ctypes.c_int64(N),
                              ctypes.c_int32(block_size), ctypes.c_uint64(seed),
                              _p(blk_off, I64), None)
    hashes = np.zeros(max(int(NB), 1), dtype=np.uint64)
    lib().orc_block_hash(_p(tokens, I32), _p(tok_off, I64), ctypes.c_int64(N),
                         ctypes.c_int32(block_size), ctypes.c_uint64(seed),
                         _p(blk_off, I64), _p(hashes, U64))
    return blk_off, hashes[:int(NB)]


@dataclass
class Radix:
    """Flattened radix cache, SURVEY.md section 8(b) peek_radix (read-only)."""
    c_tokens: np.ndarray      # int32[CT]
    n_tok_off: np.ndarray     # int64[V]
    n_tok_len: np.ndarray     # int32[V]
    n_child_off: np.ndarray   # int32[V+1]
    e_first_tok: np.ndarray   # int32[E]
    e_child: np.ndarray       # int32[E]


def lpm_radix(tokens, tok_off, radix: Radix):
    """O2 radix mode (Alg. 1's result).  int32[N] hit in tokens."""
    tokens = _c(tokens, np.int32)
    tok_off = _c(tok_off, np.int64)
    N = tok_off.shape[0] - 1
    hit = np.zeros(N, dtype=np.int32)
    ct = _c(radix.c_tokens, np.int32)
    if ct.shape[0] == 0:
        ct = np.zeros(1, dtype=np.int32)
    ef = _c(radix.e_first_tok, np.int32)
    ec = _c(radix.e_child, np.int32)
    if ef.shape[0] == 0:
        ef = np.zeros(1, dtype=np.int32)
        ec = np.zeros(1, dtype=np.int32)
    lib().orc_lpm_radix(_p(tokens, I32), _p(tok_off, I64), ctypes.c_int64(N),
                        _p(ct, I32), _p(_c(radix.n_tok_off, np.int64), I64),
                        _p(_c(radix.n_tok_len, np.int32), I32),
                        _p(_c(radix.n_child_off, np.int32), I32),
                        _p(ef, I32), _p(ec, I32), _p(hit, I32))
    return hit


def lpm_hash(hashes, blk_off, t_keys, block_size: int = 16):
    """O2 hash mode: B * leading blocks present, first miss stops."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    t_keys = _c(t_keys, np.uint64)
    N = blk_off.shape[0] - 1
    hit = np.zeros(N, dtype=np.int32)
    lib().orc_lpm_hash(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N),
                       ctypes.c_int32(block_size), _p(t_keys, U64),
                       ctypes.c_int64(t_keys.shape[0]), _p(hit, I32))
    return hit


@dataclass
class PendingTree:
    order: np.ndarray          # int32[N] sorted position -> request
    lcp: np.ndarray            # int32[N] blocks shared by sorted neighbours j-1, j
    group_id: np.ndarray       # int32[N] by request
    group_size: np.ndarray     # int32[N] by request
    cluster_depth: np.ndarray  # int32[N] by request (blocks)
    cluster_size: np.ndarray   # int32[N] by request
    cluster_id: np.ndarray     # int64[N] by request
    n_groups: int

    @property
    def has_sharing(self) -> bool:
        """some root child has pending_count >= 2."""
        return bool(lib().orc_has_sharing(_p(self.group_size, I32),
                                          ctypes.c_int64(self.group_size.shape[0])))


def pending_tree(hashes, blk_off) -> PendingTree:
    """O3."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    N = blk_off.shape[0] - 1
    z32 = lambda: np.zeros(N, dtype=np.int32)
    t = PendingTree(z32(), z32(), z32(), z32(), z32(), z32(), np.zeros(N, dtype=np.int64), 0)
    ng = np.zeros(1, dtype=np.int32)
    lib().orc_pending_tree(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N),
                           _p(t.order, I32), _p(t.lcp, I32), _p(t.group_id, I32),
                           _p(t.group_size, I32), _p(t.cluster_depth, I32),
                           _p(t.cluster_size, I32), _p(t.cluster_id, I64), _p(ng, I32))
    t.n_groups = int(ng[0])
    return t


def demand(hashes, blk_off, t_keys):
    """O4 (Eq. 2).  int32[S]."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    t_keys = _c(t_keys, np.uint64)
    N = blk_off.shape[0] - 1
    out = np.zeros(t_keys.shape[0], dtype=np.int32)
    lib().orc_demand(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N), _p(t_keys, U64),
                     ctypes.c_int64(t_keys.shape[0]), _p(out, I32))
    return out


def clpm_order(hit, cluster_size, arrival=None):
    """O5 (sub-key of Eq. 1).  int32[N] permutation."""
    hit = _c(hit, np.int32)
    cluster_size = _c(cluster_size, np.int32)
    arr = None if arrival is None else _c(arrival, np.int32)
    N = hit.shape[0]
    out = np.zeros(N, dtype=np.int32)
    lib().orc_clpm_order(_p(hit, I32), _p(cluster_size, I32), _p(arr, I32),
                         ctypes.c_int64(N), _p(out, I32))
    return out


def score(hashes, blk_off, block_size: int = 16):
    """O6 ancestor score.  int64[N]."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    N = blk_off.shape[0] - 1
    out = np.zeros(N, dtype=np.int64)
    lib().orc_score(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N), ctypes.c_int32(block_size),
                    _p(out, I64))
    return out


def evict_score(hashes, blk_off, t_keys, block_size: int = 16):
    """O7 eviction score per table slot (Eq. 2).  int64[S]."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    t_keys = _c(t_keys, np.uint64)
    N = blk_off.shape[0] - 1
    out = np.zeros(t_keys.shape[0], dtype=np.int64)
    lib().orc_evict_score(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N), ctypes.c_int32(block_size),
                          _p(t_keys, U64), ctypes.c_int64(t_keys.shape[0]), _p(out, I64))
    return out


def sections(hashes, blk_off, hit, tau: int = 0, arrival=None):
    """O8 warm / pioneer / sibling (Alg. 2).  int32[N] in {0, 1, 2}."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    hit = _c(hit, np.int32)
    arr = None if arrival is None else _c(arrival, np.int32)
    N = blk_off.shape[0] - 1
    out = np.zeros(N, dtype=np.int32)
    lib().orc_sections(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N), _p(hit, I32),
                       ctypes.c_int32(tau), _p(arr, I32), _p(out, I32))
    return out


def clpm_order_full(section, hit, score_, cluster_size, arrival=None):
    """O9 the full Eq. 1 key.  int32[N] permutation."""
    section = _c(section, np.int32)
    hit = _c(hit, np.int32)
    score_ = _c(score_, np.int64)
    cluster_size = _c(cluster_size, np.int32)
    arr = None if arrival is None else _c(arrival, np.int32)
    N = hit.shape[0]
    out = np.zeros(N, dtype=np.int32)
    lib().orc_clpm_order_full(_p(section, I32), _p(hit, I32), _p(score_, I64), _p(cluster_size, I32),
                              _p(arr, I32), ctypes.c_int64(N), _p(out, I32))
    return out


def group_major(lane_order, cluster_id):
    """O10 group-major admission order (worked example PAPER.md:55).  int32[N]."""
    lane_order = _c(lane_order, np.int32)
    cluster_id = _c(cluster_id, np.int64)
    N = lane_order.shape[0]
    out = np.zeros(N, dtype=np.int32)
    lib().orc_group_major(_p(lane_order, I32), _p(cluster_id, I64), ctypes.c_int64(N), _p(out, I32))
    return out


def offline_phase1(hashes, blk_off, depth_blocks: int = 8):
    """O11 PEEK-offline phase 1.  Returns (order int32[N],
    guards float64[4] = duplication, coverage, mean sharing depth in tokens, fired)."""
    hashes = _c(hashes, np.uint64)
    if hashes.shape[0] == 0:
        hashes = np.zeros(1, dtype=np.uint64)
    blk_off = _c(blk_off, np.int64)
    N = blk_off.shape[0] - 1
    out = np.zeros(N, dtype=np.int32)
    guards = np.zeros(4, dtype=np.float64)
    lib().orc_offline_phase1(_p(hashes, U64), _p(blk_off, I64), ctypes.c_int64(N), ctypes.c_int32(depth_blocks),
                             _p(out, I32), guards.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return out, guards


def radix_demand(tokens, tok_off, radix: Radix):
    """O12 per-radix-node pending demand (R26).  int32[V], node 0 (root) = N."""
    tokens = _c(tokens, np.int32)
    if tokens.shape[0] == 0:
        tokens = np.zeros(1, dtype=np.int32)
    tok_off = _c(tok_off, np.int64)
    N = tok_off.shape[0] - 1
    V = radix.n_tok_len.shape[0]
    out = np.zeros(V, dtype=np.int32)
    e_first = radix.e_first_tok if radix.e_first_tok.shape[0] else np.zeros(1, np.int32)
    e_child = radix.e_child if radix.e_child.shape[0] else np.zeros(1, np.int32)
    c_tok = radix.c_tokens if radix.c_tokens.shape[0] else np.zeros(1, np.int32)
    lib().orc_radix_demand(_p(tokens, I32), _p(tok_off, I64), ctypes.c_int64(N), _p(_c(c_tok, np.int32), I32),
                           _p(_c(radix.n_tok_off, np.int64), I64), _p(_c(radix.n_tok_len, np.int32), I32),
                           _p(_c(radix.n_child_off, np.int32), I32), _p(_c(e_first, np.int32), I32),
                           _p(_c(e_child, np.int32), I32), ctypes.c_int32(V), _p(out, I32))
    return out


def lane_b(section, hit, arrival=None):
    """O13 fairness lane order (Alg. 2 line 18).  int32[N]."""
    section = _c(section, np.int32)
    hit = _c(hit, np.int32)
    arr = None if arrival is None else _c(arrival, np.int32)
    N = hit.shape[0]
    out = np.zeros(N, dtype=np.int32)
    lib().orc_lane_b(_p(section, I32), _p(hit, I32), _p(arr, I32), ctypes.c_int64(N), _p(out, I32))
    return out


def dynamic_lane(cluster_size, age_pressure: float, prev: float):
    """O14 dynamic-lane controller.  Returns (new 1 - alpha, singleton_frac)."""
    cluster_size = _c(cluster_size, np.int32)
    out = np.zeros(2, dtype=np.float64)
    lib().orc_dynamic_lane(_p(cluster_size, I32), ctypes.c_int64(cluster_size.shape[0]),
                           ctypes.c_double(age_pressure), ctypes.c_double(prev),
                           out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return float(out[0]), float(out[1])


def stride_interleave(lane_a, lane_b, alpha: float):
    """O15 stride interleave of the two lanes (Alg. 2 line 22; R28).  int32[N]."""
    lane_a = _c(lane_a, np.int32)
    lane_b = _c(lane_b, np.int32)
    N = lane_a.shape[0]
    out = np.zeros(N, dtype=np.int32)
    lib().orc_stride_interleave(_p(lane_a, I32), _p(lane_b, I32), ctypes.c_int64(N), ctypes.c_double(alpha),
                                _p(out, I32))
    return out
