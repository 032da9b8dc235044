"""Thin ctypes binding over libpeek.so (include/peek.h): argument marshalling only.

Same four names as the C ABI.  PyTorch supplies device memory and the current CUDA stream; every
step of the path runs in the library's kernels.  There is no fallback: if libpeek.so is missing or
a call fails, this module raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# PEEK_LIB selects another build of the same library (the checked build, a traced build)
LIB_PATH = os.environ.get("PEEK_LIB") or os.path.join(_HERE, "libpeek.so")
_lib = None

CALL_BLOCK_HASH, CALL_LPM, CALL_PENDING_TREE, CALL_DEMAND_RANK = 0, 1, 2, 3
CALL_CLPM_SIGNALS, CALL_CLPM_ORDER_FULL, CALL_CLPM_GROUP_MAJOR, CALL_OFFLINE_PHASE1 = 4, 5, 6, 7
CALL_PENDING_TREE_UPDATE = 8
EXPORTS = ["peek_status_string", "peek_last_error", "peek_version", "peek_workspace_bytes",
           "peek_profile_enable", "peek_profile_slots", "peek_profile_name", "peek_profile_read",
           "peek_launch_count", "peek_set_option", "peek_lpm_counters",
           "peek_block_hash", "peek_block_hash_static", "peek_lpm", "peek_pending_tree", "peek_demand_rank",
           "peek_clpm_signals", "peek_clpm_order_full", "peek_clpm_group_major", "peek_offline_phase1", "peek_radix_demand",
           "peek_clpm_lane_b", "peek_dynamic_lane", "peek_pending_tree_update",
           "peek_stride_interleave"]


class PeekError(RuntimeError):
    pass


class _Radix(ctypes.Structure):
    _fields_ = [("c_tokens", ctypes.c_void_p), ("CT", ctypes.c_int64),
                ("n_tok_off", ctypes.c_void_p), ("n_tok_len", ctypes.c_void_p),
                ("n_child_off", ctypes.c_void_p), ("V", ctypes.c_int32),
                ("e_first_tok", ctypes.c_void_p), ("e_child", ctypes.c_void_p),
                ("E", ctypes.c_int32)]


class _Table(ctypes.Structure):
    _fields_ = [("t_keys", ctypes.c_void_p), ("S", ctypes.c_int64)]


class _TreeView(ctypes.Structure):
    _fields_ = [("order", ctypes.c_void_p), ("lcp", ctypes.c_void_p)]


def lib():
    """Load libpeek.so; raise loudly if it has not been built (python -m paper_2607_02525_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PeekError("libpeek.so not found at %s: build it with "
                            "`python -m paper_2607_02525_b200.build` (no CPU fallback exists)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32, u64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_uint64
        L.peek_status_string.restype = ctypes.c_char_p
        L.peek_status_string.argtypes = [i32]
        L.peek_last_error.restype = ctypes.c_char_p
        L.peek_version.restype = i32
        L.peek_workspace_bytes.restype = i32
        L.peek_workspace_bytes.argtypes = [i32, i64, i64, i64, i64, i64, ctypes.POINTER(i64)]
        L.peek_set_option.restype = i32
        L.peek_set_option.argtypes = [i32, i64]
        L.peek_block_hash.restype = i32
        L.peek_block_hash.argtypes = [vp, vp, i64, i32, u64, vp, vp, i64, vp, i64, vp]
        L.peek_block_hash_static.restype = i32
        L.peek_block_hash_static.argtypes = [vp, vp, i64, i32, u64, vp, vp, i64, vp]
        L.peek_lpm.restype = i32
        L.peek_lpm.argtypes = [vp, vp, vp, vp, i64, i32, ctypes.POINTER(_Radix), ctypes.POINTER(_Table),
                               ctypes.POINTER(_TreeView), vp, vp, vp, i64, vp]
        L.peek_pending_tree.restype = i32
        L.peek_pending_tree.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, vp]
        L.peek_demand_rank.restype = i32
        L.peek_demand_rank.argtypes = [vp, vp, i64, vp, vp, ctypes.POINTER(_Table), vp, vp, vp, vp, vp,
                                       vp, i64, vp]
        L.peek_clpm_signals.restype = i32
        L.peek_clpm_signals.argtypes = [vp, vp, i64, vp, vp, vp, i32, vp, ctypes.POINTER(_Table), vp, vp, vp,
                                        vp, i64, vp]
        L.peek_clpm_order_full.restype = i32
        L.peek_clpm_order_full.argtypes = [vp, vp, vp, vp, vp, i64, vp, vp, i64, vp]
        L.peek_clpm_group_major.restype = i32
        L.peek_clpm_group_major.argtypes = [vp, vp, i64, vp, vp, i64, vp]
        L.peek_pending_tree_update.restype = i32
        L.peek_pending_tree_update.argtypes = [vp, vp, i64, i64, vp, vp, i64, vp] + [vp] * 8 + [vp, i64, vp]
        L.peek_stride_interleave.restype = i32
        L.peek_stride_interleave.argtypes = [vp, vp, i64, ctypes.c_double, vp, vp, i64, vp]
        L.peek_clpm_lane_b.restype = i32
        L.peek_clpm_lane_b.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp]
        L.peek_dynamic_lane.restype = i32
        L.peek_dynamic_lane.argtypes = [vp, i64, ctypes.c_double, ctypes.c_double, vp, vp, i64, vp]
        L.peek_radix_demand.restype = i32
        L.peek_radix_demand.argtypes = [vp, vp, i64, ctypes.POINTER(_Radix), vp, vp, vp]
        L.peek_offline_phase1.restype = i32
        L.peek_offline_phase1.argtypes = [vp, vp, i64, i32, vp, vp, vp, i64, vp]
        _lib = L
    return _lib


def _check(st: int, what: str):
    if st != 0:
        L = lib()
        raise PeekError("%s: %s (%s)" % (what, L.peek_status_string(st).decode(),
                                         L.peek_last_error().decode()))


def _ptr(t: Optional[torch.Tensor], dtype=None):
    if t is None:
        return None
    if not t.is_cuda:
        raise PeekError("expected a CUDA tensor (the library has no CPU path)")
    if not t.is_contiguous():
        raise PeekError("expected a contiguous tensor")
    if dtype is not None and t.dtype != dtype:
        raise PeekError("expected dtype %s, got %s" % (dtype, t.dtype))
    return ctypes.c_void_p(t.data_ptr())


_dummies = {}


def _hptr(t: Optional[torch.Tensor]):
    """Pointer to a hash array.  A queue without a single full block has NB = 0 and an empty tensor,
    whose data pointer is NULL; the library wants a non-NULL `hashes` whenever an output needs the
    chains, so such a tensor is passed as a one-element dummy that is never read."""
    if t is None:
        return None
    if t.numel() == 0:
        key = (t.device.type, t.device.index)
        if key not in _dummies:
            _dummies[key] = torch.zeros(1, dtype=U64, device=t.device)
        return _ptr(_dummies[key])
    return _ptr(t, U64)


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


_ws_cache = {}


def workspace_bytes(call_id: int, N=0, T=0, NB=0, S=0, V=0) -> int:
    out = ctypes.c_int64(0)
    _check(lib().peek_workspace_bytes(call_id, N, T, NB, S, V, ctypes.byref(out)), "peek_workspace_bytes")
    return int(out.value)


def _ws(call_id, device, **sizes):
    """Scratch for one call, cached per (device, stream, call): two streams never share a buffer."""
    if torch.device(device).type != "cuda":
        raise PeekError("expected CUDA tensors (the library has no CPU path)")
    need = workspace_bytes(call_id, **sizes)
    key = (str(device), int(torch.cuda.current_stream(device).cuda_stream), call_id)
    buf = _ws_cache.get(key)
    if buf is None or buf.numel() < need:
        buf = torch.empty(need, dtype=torch.uint8, device=device)
        _ws_cache[key] = buf
    return buf, need


U64 = torch.uint64


@dataclass
class Radix:
    """Flattened radix cache on the device (include/peek.h peek_radix)."""
    c_tokens: torch.Tensor     # int32[CT]
    n_tok_off: torch.Tensor    # int64[V]
    n_tok_len: torch.Tensor    # int32[V]
    n_child_off: torch.Tensor  # int32[V+1]
    e_first_tok: torch.Tensor  # int32[E]
    e_child: torch.Tensor      # int32[E]

    def _c(self) -> _Radix:
        V = int(self.n_tok_len.shape[0])
        E = int(self.e_child.shape[0])
        return _Radix(_ptr(self.c_tokens, torch.int32) if self.c_tokens.numel() else None,
                      int(self.c_tokens.shape[0]), _ptr(self.n_tok_off, torch.int64),
                      _ptr(self.n_tok_len, torch.int32), _ptr(self.n_child_off, torch.int32), V,
                      _ptr(self.e_first_tok, torch.int32) if E else None,
                      _ptr(self.e_child, torch.int32) if E else None, E)


@dataclass
class PendingTree:
    order: torch.Tensor
    lcp: torch.Tensor
    group_id: torch.Tensor
    group_size: torch.Tensor
    cluster_depth: torch.Tensor
    cluster_size: torch.Tensor
    cluster_id: torch.Tensor
    n_groups: torch.Tensor  # int32[1] on the device


def peek_block_hash(tokens: torch.Tensor, tok_off: torch.Tensor, NB: int, block_size: int = 16,
                    seed: int = 0, blk_off: Optional[torch.Tensor] = None,
                    hashes: Optional[torch.Tensor] = None):
    """a1.  NB = sum floor(len_r / block_size), computed by the caller from its
    host copy of tok_off.  Returns (blk_off int64[N+1], hashes uint64[NB])."""
    N = int(tok_off.shape[0]) - 1
    dev = tok_off.device
    if blk_off is None:
        blk_off = torch.empty(N + 1, dtype=torch.int64, device=dev)
    if hashes is None:
        hashes = torch.empty(max(NB, 1), dtype=U64, device=dev)
    ws, nbytes = _ws(CALL_BLOCK_HASH, dev, N=N)
    st = lib().peek_block_hash(_ptr(tokens, torch.int32) if tokens.numel() else None,
                               _ptr(tok_off, torch.int64), N, block_size, ctypes.c_uint64(seed),
                               _ptr(blk_off, torch.int64), _ptr(hashes, U64), NB, _ptr(ws), nbytes, _stream())
    _check(st, "peek_block_hash")
    return blk_off, hashes[:NB]


BLOCK_HASH_STATIC_MAX_N = 4194304  # include/peek.h PEEK_BLOCK_HASH_STATIC_MAX_N


def peek_block_hash_static(tokens: torch.Tensor, tok_off: torch.Tensor, NB: int, blk_off: torch.Tensor,
                           hashes: torch.Tensor, block_size: int = 16, seed: int = 0):
    """peek_block_hash without a workspace: the scratch is a static device array inside the library
    (at most BLOCK_HASH_STATIC_MAX_N requests; calls that overlap on the GPU race).  Nothing is
    allocated here either: the caller passes both outputs.  Returns (blk_off, hashes[:NB])."""
    N = int(tok_off.shape[0]) - 1
    st = lib().peek_block_hash_static(_ptr(tokens, torch.int32) if tokens.numel() else None,
                                      _ptr(tok_off, torch.int64), N, block_size, ctypes.c_uint64(seed),
                                      _ptr(blk_off, torch.int64), _ptr(hashes, U64), NB, _stream())
    _check(st, "peek_block_hash_static")
    return blk_off, hashes[:NB]


def peek_pending_tree(hashes: torch.Tensor, blk_off: torch.Tensor, signals: bool = True) -> PendingTree:
    """a2-a4."""
    N = int(blk_off.shape[0]) - 1
    dev = blk_off.device
    e32 = lambda: torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    t = PendingTree(e32(), e32(), e32(), e32(), e32(), e32(),
                    torch.empty(max(N, 1), dtype=torch.int64, device=dev)[:N],
                    torch.zeros(1, dtype=torch.int32, device=dev))
    ws, nbytes = _ws(CALL_PENDING_TREE, dev, N=N)
    sig = (lambda x: _ptr(x)) if signals else (lambda x: None)
    st = lib().peek_pending_tree(_hptr(hashes), _ptr(blk_off, torch.int64),
                                 N, _ptr(t.order), _ptr(t.lcp), sig(t.group_id), sig(t.group_size),
                                 sig(t.cluster_depth), sig(t.cluster_size), sig(t.cluster_id),
                                 sig(t.n_groups), _ptr(ws), nbytes, _stream())
    _check(st, "peek_pending_tree")
    return t


def peek_lpm(tokens=None, tok_off=None, hashes=None, blk_off=None, radix: Optional[Radix] = None,
             t_keys: Optional[torch.Tensor] = None, tree: Optional[PendingTree] = None,
             block_size: int = 16, want_radix: Optional[bool] = None, want_hash: Optional[bool] = None):
    """a5/a6 (Alg. 1).  Returns (hit_radix | None, hit_hash | None)."""
    ref = tok_off if tok_off is not None else blk_off
    N = int(ref.shape[0]) - 1
    dev = ref.device
    want_radix = radix is not None if want_radix is None else want_radix
    want_hash = t_keys is not None if want_hash is None else want_hash
    hr = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N] if want_radix else None
    hh = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N] if want_hash else None
    cr = radix._c() if radix is not None else None
    ct = _Table(_ptr(t_keys, U64), int(t_keys.shape[0])) if t_keys is not None else None
    cv = _TreeView(_ptr(tree.order, torch.int32), _ptr(tree.lcp, torch.int32)) if tree is not None else None
    ws, nbytes = _ws(CALL_LPM, dev, N=N, V=max(int(radix.n_tok_len.shape[0]), int(radix.e_child.shape[0])) if radix is not None else 0)
    if tokens is not None and tokens.numel() == 0:  # all requests empty: still a valid pointer
        tokens = torch.zeros(4, dtype=torch.int32, device=dev)
    st = lib().peek_lpm(_ptr(tokens), _ptr(tok_off),
                        _hptr(hashes), _ptr(blk_off), N,
                        block_size, ctypes.byref(cr) if cr is not None else None,
                        ctypes.byref(ct) if ct is not None else None,
                        ctypes.byref(cv) if cv is not None else None, _ptr(hr), _ptr(hh), _ptr(ws), nbytes,
                        _stream())
    _check(st, "peek_lpm")
    return hr, hh


def peek_demand_rank(hashes=None, blk_off=None, tree: Optional[PendingTree] = None,
                     t_keys: Optional[torch.Tensor] = None, hit: Optional[torch.Tensor] = None,
                     cluster_size: Optional[torch.Tensor] = None, arrival: Optional[torch.Tensor] = None,
                     want_demand: Optional[bool] = None, want_order: Optional[bool] = None):
    """a7/a8 (Eq. 1).  Returns (demand | None, clpm_order | None)."""
    ref = blk_off if blk_off is not None else hit
    N = int(ref.shape[0]) - (1 if blk_off is not None else 0)
    dev = ref.device
    want_demand = t_keys is not None if want_demand is None else want_demand
    want_order = hit is not None if want_order is None else want_order
    S = int(t_keys.shape[0]) if t_keys is not None else 0
    demand = torch.empty(S, dtype=torch.int32, device=dev) if want_demand else None
    out = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N] if want_order else None
    ct = _Table(_ptr(t_keys, U64), S) if t_keys is not None else None
    ws, nbytes = _ws(CALL_DEMAND_RANK, dev, N=N, S=S)
    st = lib().peek_demand_rank(_hptr(hashes),
                                _ptr(blk_off), N, _ptr(tree.order) if tree is not None else None,
                                _ptr(tree.lcp) if tree is not None else None,
                                ctypes.byref(ct) if ct is not None else None, _ptr(hit), _ptr(cluster_size),
                                _ptr(arrival), _ptr(demand), _ptr(out), _ptr(ws), nbytes, _stream())
    _check(st, "peek_demand_rank")
    return demand, out


def peek_clpm_signals(hashes, blk_off, tree: PendingTree, hit: Optional[torch.Tensor] = None, tau: int = 0,
                      arrival: Optional[torch.Tensor] = None, t_keys: Optional[torch.Tensor] = None,
                      want_section: Optional[bool] = None, want_score: bool = True,
                      want_evict: Optional[bool] = None):
    """a9.
    Returns (section int32[N] | None, score int64[N] | None, evict_score int64[S] | None)."""
    N = int(blk_off.shape[0]) - 1
    dev = blk_off.device
    want_section = hit is not None if want_section is None else want_section
    want_evict = t_keys is not None if want_evict is None else want_evict
    S = int(t_keys.shape[0]) if t_keys is not None else 0
    section = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N] if want_section else None
    score = torch.empty(max(N, 1), dtype=torch.int64, device=dev)[:N] if want_score else None
    evict = torch.empty(S, dtype=torch.int64, device=dev) if want_evict else None
    ct = _Table(_ptr(t_keys, U64), S) if t_keys is not None else None
    ws, nbytes = _ws(CALL_CLPM_SIGNALS, dev, N=N, S=S)
    st = lib().peek_clpm_signals(_hptr(hashes), _ptr(blk_off), N,
                                 _ptr(tree.order), _ptr(tree.lcp), _ptr(hit), int(tau), _ptr(arrival),
                                 ctypes.byref(ct) if ct is not None else None, _ptr(section), _ptr(score),
                                 _ptr(evict), _ptr(ws), nbytes, _stream())
    _check(st, "peek_clpm_signals")
    return section, score, evict


def peek_clpm_order_full(section, hit, score, cluster_size, arrival=None):
    """a10: the five-part key of Eq. 1.  int32[N] permutation."""
    N = int(hit.shape[0])
    dev = hit.device
    out = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    ws, nbytes = _ws(CALL_CLPM_ORDER_FULL, dev, N=N)
    st = lib().peek_clpm_order_full(_ptr(section), _ptr(hit), _ptr(score), _ptr(cluster_size), _ptr(arrival), N,
                                    _ptr(out), _ptr(ws), nbytes, _stream())
    _check(st, "peek_clpm_order_full")
    return out


def peek_clpm_group_major(lane_order, cluster_id):
    """a11: group-major admission order.  int32[N] permutation."""
    N = int(lane_order.shape[0])
    dev = lane_order.device
    out = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    ws, nbytes = _ws(CALL_CLPM_GROUP_MAJOR, dev, N=N)
    st = lib().peek_clpm_group_major(_ptr(lane_order), _ptr(cluster_id), N, _ptr(out), _ptr(ws), nbytes, _stream())
    _check(st, "peek_clpm_group_major")
    return out


def peek_pending_tree_update(hashes, blk_off, M: int, old: PendingTree, remap, signals: bool = True) -> PendingTree:
    """a13: incremental maintenance.  hashes / blk_off describe the NEW queue
    (survivors renumbered by remap, then M arrivals); returns what peek_pending_tree would."""
    N = int(blk_off.shape[0]) - 1
    N_old = int(old.order.shape[0])
    dev = blk_off.device
    i32 = lambda: torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    t = PendingTree(i32(), i32(), i32() if signals else None, i32() if signals else None,
                    i32() if signals else None, i32() if signals else None,
                    torch.empty(max(N, 1), dtype=torch.int64, device=dev)[:N] if signals else None,
                    torch.zeros(1, dtype=torch.int32, device=dev) if signals else None)
    L = lib()
    nb = ctypes.c_int64(0)
    _check(L.peek_workspace_bytes(CALL_PENDING_TREE_UPDATE, N, N_old, int(M), 0, 0, ctypes.byref(nb)), "peek_workspace_bytes")
    ws = torch.empty(max(int(nb.value), 256), dtype=torch.uint8, device=dev)
    st = L.peek_pending_tree_update(_hptr(hashes), _ptr(blk_off),
                                    N, int(M), _ptr(old.order), _ptr(old.lcp), N_old, _ptr(remap),
                                    _ptr(t.order), _ptr(t.lcp), _ptr(t.group_id), _ptr(t.group_size),
                                    _ptr(t.cluster_depth), _ptr(t.cluster_size), _ptr(t.cluster_id), _ptr(t.n_groups),
                                    _ptr(ws), int(nb.value), _stream())
    _check(st, "peek_pending_tree_update")
    return t


def peek_stride_interleave(lane_a, lane_b, alpha: float = 0.7):
    """a11d: stride interleave of the two lanes (Alg. 2 line 22; R28).  int32[N]."""
    N = int(lane_a.shape[0])
    dev = lane_a.device
    out = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    nbytes = max(256, (N + 31) // 32 * 4)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    st = lib().peek_stride_interleave(_ptr(lane_a), _ptr(lane_b), N, float(alpha), _ptr(out), _ptr(ws), nbytes, _stream())
    _check(st, "peek_stride_interleave")
    return out


def peek_clpm_lane_b(section, hit, arrival=None):
    """a11b: fairness lane order (Alg. 2 line 18).  int32[N] permutation."""
    N = int(hit.shape[0])
    dev = hit.device
    out = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    ws, nbytes = _ws(CALL_CLPM_ORDER_FULL, dev, N=N)
    st = lib().peek_clpm_lane_b(_ptr(section), _ptr(hit), _ptr(arrival), N, _ptr(out), _ptr(ws), nbytes, _stream())
    _check(st, "peek_clpm_lane_b")
    return out


def peek_dynamic_lane(cluster_size, age_pressure: float, prev_fair_share: float):
    """a11c: dynamic-lane controller.  float64[2] on the device:
    (new fairness share 1 - alpha, singleton_frac)."""
    N = int(cluster_size.shape[0])
    dev = cluster_size.device
    out = torch.zeros(2, dtype=torch.float64, device=dev)
    ws = torch.empty(256, dtype=torch.uint8, device=dev)
    st = lib().peek_dynamic_lane(_ptr(cluster_size), N, float(age_pressure), float(prev_fair_share), _ptr(out),
                                 _ptr(ws), 256, _stream())
    _check(st, "peek_dynamic_lane")
    return out


def peek_radix_demand(tokens, tok_off, radix: Radix, hit_radix):
    """a9b: per-radix-node pending demand (R26).  int32[V], node 0 = N."""
    N = int(tok_off.shape[0]) - 1
    V = int(radix.n_tok_len.shape[0])
    out = torch.empty(V, dtype=torch.int32, device=tok_off.device)
    cr = radix._c()
    if tokens is not None and tokens.numel() == 0:  # all requests empty: still a valid pointer
        tokens = torch.zeros(4, dtype=torch.int32, device=tok_off.device)
    st = lib().peek_radix_demand(_ptr(tokens), _ptr(tok_off), N,
                                 ctypes.byref(cr), _ptr(hit_radix), _ptr(out), _stream())
    _check(st, "peek_radix_demand")
    return out


def peek_offline_phase1(hashes, blk_off, depth_blocks: int = 8):
    """a12: PEEK-offline phase 1.  Returns (order int32[N],
    guards float64[4] on the device: duplication, coverage, mean sharing depth in tokens, fired)."""
    N = int(blk_off.shape[0]) - 1
    dev = blk_off.device
    order = torch.empty(max(N, 1), dtype=torch.int32, device=dev)[:N]
    guards = torch.zeros(4, dtype=torch.float64, device=dev)
    ws, nbytes = _ws(CALL_OFFLINE_PHASE1, dev, N=N)
    st = lib().peek_offline_phase1(_hptr(hashes), _ptr(blk_off),
                                   N, int(depth_blocks), _ptr(order), _ptr(guards), _ptr(ws), nbytes, _stream())
    _check(st, "peek_offline_phase1")
    return order, guards


OPT_LPM_STRATEGY, OPT_LPM_WINDOW, OPT_GRID_LIMIT, OPT_TREE_LOCAL_CAP = 1, 2, 3, 4
LPM_AUTO, LPM_DUAL_WALK, LPM_SPECULATIVE = 0, 1, 2


def lpm_counters(buf: Optional[torch.Tensor]):
    """peek_lpm_counters: uint64[4] device tensor that later peek_lpm calls add to, or None (off)."""
    L = lib()
    L.peek_lpm_counters.restype = ctypes.c_int32
    L.peek_lpm_counters.argtypes = [ctypes.c_void_p]
    _check(L.peek_lpm_counters(_ptr(buf) if buf is not None else None), "peek_lpm_counters")


def set_option(key: int, value: int) -> None:
    """include/peek.h "options": tuning and test hooks; results never depend on them."""
    _check(lib().peek_set_option(key, value), "peek_set_option")


# ---- tracing (include/peek.h "tracing") ---------------------------------------------------
def profile_enable(on: bool) -> None:
    L = lib()
    L.peek_profile_enable.argtypes = [ctypes.c_int32]
    L.peek_profile_enable(1 if on else 0)


def profile_read(reset: bool = True) -> dict:
    """{slot name: (total_ms, groups)} for the kernel groups recorded since the last reset."""
    L = lib()
    L.peek_profile_name.restype = ctypes.c_char_p
    L.peek_profile_name.argtypes = [ctypes.c_int32]
    L.peek_profile_read.restype = ctypes.c_int32
    L.peek_profile_read.argtypes = [ctypes.c_int32, ctypes.POINTER(ctypes.c_double),
                                    ctypes.POINTER(ctypes.c_int64), ctypes.c_int32]
    out = {}
    for s in range(int(L.peek_profile_slots())):
        ms, n = ctypes.c_double(0), ctypes.c_int64(0)
        _check(L.peek_profile_read(s, ctypes.byref(ms), ctypes.byref(n), 1 if reset else 0), "peek_profile_read")
        out[L.peek_profile_name(s).decode()] = (float(ms.value), int(n.value))
    return out


def launch_count() -> int:
    L = lib()
    L.peek_launch_count.restype = ctypes.c_int64
    return int(L.peek_launch_count())
