#!/usr/bin/env python
"""bench.py — one JSON line for the PEEK hot path on B200 (contract in DESIGN.md "Measurement").

A step = one pass of the whole hot path over one batch of pending requests, through the C ABI:
peek_block_hash -> peek_pending_tree -> peek_lpm (radix + hash mode, co-descent) ->
peek_demand_rank.  Default workload: BASELINE.json configs[4] (agentic multi-turn, 1 048 576
pending requests, ~4.3e9 tokens), the "largest config" north_star's target is quoted on.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl peek|reference]

--gpus N > 1 without a torchrun environment re-launches itself under torch.distributed.run with N
ranks (one GPU each, NCCL); every rank owns an independent batch.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from harness import workloads as W  # noqa: E402

METRIC = "lpm_queries_per_s"
UNIT = "queries/s"
CONFIG_NAMES = {1: "configs[0] tiny_shared_prompt_chat", 2: "configs[1] shared_prompt_chat_at_scale",
                3: "configs[2] long_prefix_rag", 4: "configs[3] singleton_chat_table_only",
                5: "configs[4] agentic_multi_turn_at_scale"}
PAIR_SLOTS = ("tree.persistent", "lpm.radix_walk", "lpm.hash_probe", "lpm.dual_walk")  # north_star: peek_pending_tree + peek_lpm


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def parse(argv=None):
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=20)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--config", type=int, default=5)
    p.add_argument("--seed", type=int, default=42)
    p.add_argument("--impl", default="peek", choices=["peek", "reference"])
    p.add_argument("--small", action="store_true", help="reduced sizes (tests)")
    p.add_argument("--e2e-steps", type=int, default=2)
    p.add_argument("--no-e2e", action="store_true")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--no-per-config", action="store_true", help="skip the timing of the other configs")
    p.add_argument("--no-cycle", action="store_true", help="skip the steady-state cycle measurement")
    p.add_argument("--cpu-seconds", type=float, default=15.0)
    return p.parse_args(argv)


def respawn_under_torchrun(args) -> int:
    """--gpus N > 1 outside torchrun: start N ranks of this script (one per GPU) and relay their output."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    log("[bench] --gpus %d: launching %s" % (args.gpus, " ".join(cmd)))
    return subprocess.call(cmd)


# ------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v == "Active":
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------
# inputs
# ------------------------------------------------------------------------------------------
class Inputs:
    pass


def rank_seed(seed: int, rank: int) -> int:
    """Each rank owns an independent batch: its own generator seed."""
    return seed + 1000 * rank


def max_over_ranks(ms: float, device, world: int) -> float:
    """Device time of a multi-GPU step is the max over ranks (all-reduce MAX; a no-op at world 1)."""
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: int, world: int, steps: int, ms: float) -> float:
    """Whole-job units/s: every rank processes its own batch in the same (max) time."""
    return world * units_per_rank * steps / (ms * 1e-3)


def gpu_hash_fn(dev):
    """hash_fn for workloads.build_cache: the CUDA call (the product path never touches oracle/)."""
    from paper_2607_02525_b200 import binding as B

    def fn(toks, off):
        nb = int((np.diff(off) // 16).sum())
        t = torch.from_numpy(np.ascontiguousarray(toks)).to(dev)
        o = torch.from_numpy(np.ascontiguousarray(off)).to(dev)
        bo, h = B.peek_block_hash(t, o, nb)
        torch.cuda.synchronize()
        return bo.cpu().numpy(), h.cpu().view(torch.int64).numpy().view(np.uint64)
    return fn


def upload_cache(inp, cache, dev):
    from paper_2607_02525_b200 import binding as B
    up = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    inp.cache = cache
    inp.radix = None
    if cache.radix is not None:
        r = cache.radix
        inp.radix = B.Radix(up(r.c_tokens), up(r.n_tok_off), up(r.n_tok_len), up(r.n_child_off),
                            up(r.e_first_tok), up(r.e_child))
    inp.keys = up(cache.t_keys.view(np.int64)).view(torch.uint64)
    inp.S = int(cache.t_keys.shape[0])


def build_inputs(cfg: int, seed: int, small: bool, dev) -> Inputs:
    t0 = time.time()
    wl = W.make(cfg, seed=seed, small=small)
    inp = Inputs()
    inp.cfg = cfg
    inp.wl = wl
    inp.N = wl.N
    lens = wl.queue.seq_lens()
    inp.T = int(lens.sum())
    inp.NB = int((lens // 16).sum())
    inp.tok, inp.off = wl.queue.materialize(dev)
    log("[bench] config %d: N=%d T=%d NB=%d generated+uploaded in %.1fs" % (cfg, inp.N, inp.T, inp.NB, time.time() - t0))
    t0 = time.time()
    upload_cache(inp, W.build_cache(wl, gpu_hash_fn(dev)), dev)
    inp.arrival = torch.from_numpy(np.ascontiguousarray(wl.arrival)).to(dev)
    inp.bo_buf = torch.empty(inp.N + 1, dtype=torch.int64, device=dev)
    inp.h_buf = torch.empty(max(inp.NB, 1), dtype=torch.uint64, device=dev)
    log("[bench] cache: V=%s keys=%d S=%d built in %.1fs" % (
        inp.cache.radix.V if inp.cache.radix is not None else None, inp.cache.n_keys, inp.S, time.time() - t0))
    return inp


def step(inp, tok=None, off=None):
    """One pass of the hot path; every stage is a libpeek.so call."""
    from paper_2607_02525_b200 import binding as B
    tok = inp.tok if tok is None else tok
    off = inp.off if off is None else off
    bo, h = B.peek_block_hash(tok, off, inp.NB, blk_off=inp.bo_buf, hashes=inp.h_buf)
    tree = B.peek_pending_tree(h, bo)
    hr, hh = B.peek_lpm(tok, off, h, bo, radix=inp.radix, t_keys=inp.keys, tree=tree)
    hit = hr if hr is not None else hh
    dem, order = B.peek_demand_rank(h, bo, tree=tree, t_keys=inp.keys, hit=hit,
                                    cluster_size=tree.cluster_size, arrival=inp.arrival)
    return dict(bo=bo, h=h, tree=tree, hit_radix=hr, hit_hash=hh, hit=hit, demand=dem, clpm=order)


def algorithmic_bytes(inp, out: dict) -> dict:
    """SURVEY.md section 8(d) B_alg per call, from by-products of one step (reporting only)."""
    N, T, NB, S = inp.N, inp.T, inp.NB, inp.S
    tree = out["tree"]
    order = tree.order.long()
    lcp = tree.lcp.long()
    nb = (out["bo"][1:] - out["bo"][:-1])[order]
    res = {"hash": 4 * T + 8 * NB + 16 * N, "hash.nb_scan": 24 * N}
    lc = torch.minimum(16 * (lcp + 1), 64 * torch.ceil(torch.log2(nb.double() + 2)).long()).sum().item()
    res["tree"] = int(32 * N + 192 * N + lc + 32 * N)
    U = int((nb - lcp).sum().item())
    for name, key in (("lpm.radix", "hit_radix"), ("lpm.hash", "hit_hash")):
        if out[key] is None:
            continue
        hs = out[key].long()[order]
        prev = torch.cat([torch.zeros(1, dtype=torch.long, device=hs.device), hs[:-1]])
        R = int(((prev // 16 >= lcp) | (lcp == 0)).sum().item())
        if name == "lpm.radix":
            ht = int(torch.clamp(hs - 16 * lcp, min=0).sum().item())
            res[name] = 8 * ht + 96 * R + 16 * N
        else:
            hb = int(torch.clamp(hs // 16 - lcp, min=0).sum().item())
            res[name] = 40 * (hb + R) + 16 * N
    if "lpm.radix" in res and "lpm.hash" in res:  # both modes side by side (one profile slot)
        res["lpm.both"] = res["lpm.radix"] + res["lpm.hash"]
    dplus = int((out["demand"] > 0).sum().item()) if out["demand"] is not None else 0
    res["demand"] = 40 * U + 32 * dplus + 4 * S
    res["rank"] = 208 * N
    return res


SLOT_TO_CALL = {"hash.nb_scan": "hash.nb_scan", "hash.content": "hash", "tree.persistent": "tree",
                "lpm.radix_walk": "lpm.radix", "lpm.hash_probe": "lpm.hash", "lpm.dual_walk": "lpm.both",
                "lpm.resolve_scan": None,
                "demand.count": "demand", "rank.clpm_sort": "rank"}


# ------------------------------------------------------------------------------------------
# timing
# ------------------------------------------------------------------------------------------
def time_steps(inp, steps: int, flush):
    """`steps` timed passes; flush = a buffer larger than L2 written before every pass (outside the
    event pair), or None for L2-warm passes.  Returns (ms per step list, per-slot profile, last outputs)."""
    from paper_2607_02525_b200 import binding as B
    B.profile_enable(True)
    B.profile_read(reset=True)
    evs, out = [], None
    for _ in range(steps):
        if flush is not None:
            flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = step(inp)
        e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in evs]
    prof = B.profile_read(reset=True)
    B.profile_enable(False)
    return ms, prof, out


def calls_table(inp, prof, out, steps: int, total_ms: float) -> dict:
    balg = algorithmic_bytes(inp, out)
    calls = {}
    for slot, (ms, groups) in prof.items():
        if not groups:
            continue
        per = ms / max(steps, 1)  # ms per step
        calls[slot] = {"ms_per_step": per, "share": ms / total_ms if total_ms else None}
        call = SLOT_TO_CALL.get(slot)
        if call and call in balg and per > 0:
            calls[slot]["alg_bytes"] = balg[call]
            calls[slot]["alg_GBps"] = balg[call] / (per * 1e-3) / 1e9
    return calls


def pair_summary(calls: dict, peak: float):
    """north_star: peek_lpm + peek_pending_tree against the HBM peak (algorithmic bytes / time)."""
    ms = sum(calls[s]["ms_per_step"] for s in PAIR_SLOTS if s in calls)
    by = sum(calls[s].get("alg_bytes", 0) for s in PAIR_SLOTS if s in calls)
    gbs = by / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
    return {"ms": ms, "alg_bytes": by, "alg_GBps": gbs, "frac": gbs / peak, "bar": 0.5,
            "kernels": [s for s in PAIR_SLOTS if s in calls]}


def config_summary(inp, steps: int, flush, peak: float, warm_too: bool) -> dict:
    """median / best of `steps` passes of one config; small configs also L2-warm."""
    for _ in range(3):
        step(inp)
    res = {}
    for label, fl in (("l2_flushed", flush),) + ((("l2_warm", None),) if warm_too else ()):
        ms, prof, out = time_steps(inp, steps, fl)
        tot = float(sum(ms))
        med, best = float(np.median(ms)), float(min(ms))
        sum_hit = int(out["hit"].long().sum().item())
        calls = calls_table(inp, prof, out, steps, tot)
        res[label] = {"ms_per_step_median": med, "ms_per_step_best": best,
                      "queries_per_s": inp.N / (med * 1e-3), "tokens_matched_per_s": sum_hit / (med * 1e-3),
                      "calls": {k: {"ms_per_step": v["ms_per_step"], "alg_GBps": v.get("alg_GBps")} for k, v in calls.items()},
                      "north_star_pair": pair_summary(calls, peak)}
    if inp.N <= 65536:
        # small queues are bound by launch and host latency, not by the kernels: the same step captured
        # once into a CUDA graph and replayed (what a serving loop would do), L2 warm
        try:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                step(inp)
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                gout = step(inp)
            graph.replay()
            torch.cuda.synchronize()
            ms = []
            for _ in range(steps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                graph.replay()
                e1.record()
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
            ref = step(inp)
            torch.cuda.synchronize()
            same = bool(torch.equal(gout["clpm"], ref["clpm"]) and torch.equal(gout["hit"], ref["hit"])
                        and torch.equal(gout["tree"].lcp, ref["tree"].lcp))
            med = float(np.median(ms))
            res["cuda_graph_replay"] = {"ms_per_step_median": med, "ms_per_step_best": float(min(ms)),
                                        "queries_per_s": inp.N / (med * 1e-3), "equals_eager": same}
            del graph, gout
        except Exception as e:  # capture is an optimisation of the harness, never a requirement
            res["cuda_graph_replay"] = {"error": str(e)[:200]}
    res["N"] = inp.N
    res["tokens"] = inp.T
    res["blocks"] = inp.NB
    return res


def gather_ceiling(inp, dev):
    """Random 32-byte-sector gather ceilings: the honest roofline of the probe /
    child-lookup kernels.  Over a buffer far larger than L2 (the token array, capped at 4 GiB) and
    over the table itself (8 S bytes: partly L2 resident)."""
    from harness import gather_probe as GP
    out = {}
    tok_bytes = inp.tok.numel() * 4
    big = inp.tok[: min(inp.tok.numel(), 1 << 30)] if tok_bytes >= (1 << 28) else None
    for name, buf in (("hbm", big), ("table", inp.keys)):
        if buf is None or buf.numel() * buf.element_size() < 64:
            continue
        if buf.data_ptr() % 32:
            continue
        reads = 1 << 26
        GP.random_gather(buf, reads, 1)
        torch.cuda.synchronize()
        best = None
        for it in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            GP.random_gather(buf, reads, 2 + it)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None or ms < best else best
        out[name] = {"buffer_bytes": int(buf.numel() * buf.element_size()), "reads": reads,
                     "Gsectors_per_s": reads / (best * 1e-3) / 1e9, "GBps": 32 * reads / (best * 1e-3) / 1e9}
    return out


def next_rows_timing(inp, out):
    """SURVEY.md 8(f) NEXT-1 calls (sections, ancestor score, Eq. 2 eviction score, five-part Eq. 1
    key) on the step's outputs: reported beside the step, not part of it."""
    from paper_2607_02525_b200 import binding as B
    tree, h, bo, hit = out["tree"], out["h"], out["bo"], out["hit"]

    def timed(fn, n=3):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            r = fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n, r

    ms_sig, (sec, sc, ev) = timed(lambda: B.peek_clpm_signals(h, bo, tree, hit=hit, tau=0, arrival=inp.arrival,
                                                              t_keys=inp.keys))
    ms_ord, lane = timed(lambda: B.peek_clpm_order_full(sec, hit, sc, tree.cluster_size, inp.arrival))
    ms_gm, gm = timed(lambda: B.peek_clpm_group_major(lane, tree.cluster_id))
    ms_lb, lane_b = timed(lambda: B.peek_clpm_lane_b(sec, hit, inp.arrival))
    ms_si, _ = timed(lambda: B.peek_stride_interleave(gm, lane_b, 0.7), n=1)
    ms_off, (_, guards) = timed(lambda: B.peek_offline_phase1(h, bo, 8))
    ms_nd = None
    if inp.radix is not None and out["hit_radix"] is not None:
        ms_nd, _ = timed(lambda: B.peek_radix_demand(inp.tok, inp.off, inp.radix, out["hit_radix"]))
    return {"peek_clpm_signals_ms": ms_sig, "peek_clpm_order_full_ms": ms_ord,
            "peek_clpm_group_major_ms": ms_gm, "peek_clpm_lane_b_ms": ms_lb, "peek_stride_interleave_ms": ms_si,
            "peek_offline_phase1_ms": ms_off, "peek_radix_demand_ms": ms_nd,
            "offline_guards_dup_cov_depth_fired": guards.cpu().tolist(),
            "sections_warm_pioneer_sibling": torch.bincount(sec, minlength=3).tolist()[:3]}


def work_counters(inp, out):
    """peek_lpm's work counters (PAPER.md:293 O(C x D) against O(N x D)): the dual walk over the
    tree view against the per-request walks of stock LPM, same inputs."""
    from paper_2607_02525_b200 import binding as B
    cnt = torch.zeros(4, dtype=torch.uint64, device=inp.tok.device)
    names = ("root_walks", "child_lookups", "tokens_compared", "table_probes")
    res = {}
    B.lpm_counters(cnt)
    try:
        for label, tree in (("dual_walk", out["tree"]), ("per_request", None)):
            cnt.zero_()
            B.peek_lpm(inp.tok, inp.off, out["h"], out["bo"], radix=inp.radix, t_keys=inp.keys, tree=tree)
            torch.cuda.synchronize()
            res[label] = dict(zip(names, cnt.cpu().view(torch.int64).tolist()))
    finally:
        B.lpm_counters(None)
    return res


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_source_sha(slot: str):
    """sha256 (first 12 hex digits) of the source file of the slot's kernel: stamps an ncu capture."""
    files = {"hash.content": "peek_hash.cu", "tree.persistent": "peek_tree.cu", "lpm.radix_walk": "peek_lpm.cu",
             "lpm.hash_probe": "peek_lpm.cu", "lpm.dual_walk": "peek_lpm.cu"}
    f = files.get(slot)
    if not f:
        return None
    try:
        return hashlib.sha256(open(os.path.join(ROOT, "paper_2607_02525_b200", "csrc", f), "rb").read()).hexdigest()[:12]
    except Exception:
        return None


def ncu_traffic(workload: str, slot: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of a kernel group from the
    committed ncu capture (profiles/ncu_traffic.csv: workload, slot, dram_bytes_per_launch, source_sha),
    or None when there is no capture of the kernel source as it stands (a stale number is no number)."""
    import csv
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    sha = kernel_source_sha(slot)
    try:
        for row in csv.DictReader(open(p)):
            if row["workload"] == workload and row["slot"] == slot and row.get("source_sha") == sha:
                return int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


# ------------------------------------------------------------------------------------------
# the oracle as the CPU baseline / reference arm (the only code here that touches oracle/)
# ------------------------------------------------------------------------------------------
def oracle_pass(wl, cache, n_sample: int, keep: bool = False):
    """The oracle as it stands, on the first n_sample requests of the workload against the same
    cache.  Returns (seconds for one pass of the whole path, outputs or None)."""
    import oracle
    memo = getattr(oracle_pass, "_memo", None)  # the same prefix is timed several times
    if memo is None or memo[0] is not wl or memo[1] != n_sample:
        sub = wl.queue.select(np.arange(n_sample))
        toks, off = sub.materialize_np()
        oracle_pass._memo = memo = (wl, n_sample, toks, off, np.ascontiguousarray(wl.arrival[:n_sample]))
    _, _, toks, off, arrival = memo
    radix = None
    if cache.radix is not None:
        r = cache.radix
        radix = oracle.Radix(r.c_tokens, r.n_tok_off, r.n_tok_len, r.n_child_off, r.e_first_tok, r.e_child)
    t0 = time.perf_counter()
    bo, h = oracle.block_hash(toks, off, 16, 0)
    tree = oracle.pending_tree(h, bo)
    hr = oracle.lpm_radix(toks, off, radix) if radix is not None else None
    hh = oracle.lpm_hash(h, bo, cache.t_keys)
    dem = oracle.demand(h, bo, cache.t_keys)
    clpm = oracle.clpm_order(hr if hr is not None else hh, tree.cluster_size, arrival)
    dt = time.perf_counter() - t0
    outs = dict(order=tree.order, lcp=tree.lcp, cluster_size=tree.cluster_size, hit_radix=hr, hit_hash=hh,
                demand=dem, clpm=clpm) if keep else None
    return dt, outs


def size_sample(wl, cache, budget_s: float):
    """Requests (a prefix of the workload) the oracle gets through in about budget_s seconds - the ONE
    sample rule of the cpu_baseline leg and of the reference arm.  The pass has a fixed part (the
    demand map over the whole table) and a part linear in the requests; the sample is grown from the
    measured marginal cost and is the whole queue when that fits the budget."""
    n1 = min(wl.N, 2048)
    t1, _ = oracle_pass(wl, cache, n1)
    n = n1
    if wl.N > n1:
        n2 = int(min(wl.N, max(n1 * 4, n1 * budget_s / max(t1, 1e-3) * 0.25)))
        t2, _ = oracle_pass(wl, cache, n2)
        n = n2
        marginal = max((t2 - t1) / max(n2 - n1, 1), 1e-9)
        n3 = int(min(wl.N, n2 + max(0.0, budget_s - t2) / marginal * 0.8))
        if n3 > n2 * 1.5 and t2 < 0.5 * budget_s:
            n = n3
    return n


def sample_text(n, N):
    return ("the whole queue (%d requests)" % N) if n == N else ("first %d of %d requests of the same workload" % (n, N))


def gpu_outputs_on_prefix(inp, n: int, out_full):
    """The CUDA path's outputs on the first n requests (the whole queue: the timed step's own)."""
    if n == inp.N:
        return out_full
    sub = Inputs()
    sub.__dict__.update(inp.__dict__)
    sub.N = n
    end = int(inp.off[n].item())
    sub.tok, sub.off = inp.tok[:end], inp.off[: n + 1]
    sub.NB = int(((inp.off[1: n + 1] - inp.off[:n]) // 16).sum().item())
    sub.arrival = inp.arrival[:n].contiguous()
    sub.bo_buf = torch.empty(n + 1, dtype=torch.int64, device=inp.tok.device)
    sub.h_buf = torch.empty(max(sub.NB, 1), dtype=torch.uint64, device=inp.tok.device)
    o = step(sub)
    torch.cuda.synchronize()
    return o


def parity_in_run(inp, n, orc, out_full, arrival_is_prefix_perm: bool):
    """Element-by-element comparison of the CUDA step with the oracle pass the cpu_baseline leg just
    ran (same requests, same cache): "bit-exact" or the first mismatch."""
    g = gpu_outputs_on_prefix(inp, n, out_full)
    pairs = [("order", g["tree"].order, orc["order"]), ("lcp", g["tree"].lcp, orc["lcp"]),
             ("cluster_size", g["tree"].cluster_size, orc["cluster_size"]),
             ("hit_radix", g["hit_radix"], orc["hit_radix"]), ("hit_hash", g["hit_hash"], orc["hit_hash"]),
             ("demand", g["demand"], orc["demand"]), ("clpm_order", g["clpm"], orc["clpm"])]
    checked = []
    for name, a, b in pairs:
        if a is None or b is None:
            continue
        a = a.cpu().numpy()
        if a.shape != b.shape:
            return "%s: shape %s vs %s" % (name, a.shape, b.shape)
        bad = np.nonzero(a != b)[0]
        if bad.size:
            i = int(bad[0])
            return "%s[%d]: cuda %d, oracle %d (%d of %d differ)" % (name, i, int(a[i]), int(b[i]), bad.size, a.size)
        checked.append(name)
    return "bit-exact (" + ", ".join(checked) + "; %s)" % sample_text(n, inp.N)


def cpu_inputs(cfg, seed, small):
    """Workload + cache built with the oracle's hash (reference arm: no CUDA anywhere)."""
    import oracle
    wl = W.make(cfg, seed=seed, small=small)
    cache = W.build_cache(wl, lambda t, o: oracle.block_hash(t, o, 16, 0))
    return wl, cache


def config_dict(cfg: int, small: bool, wl, cache, world: int) -> dict:
    """The `config` object of the JSON line: identical keys and values in both arms."""
    lens = wl.queue.seq_lens()
    return {"workload": CONFIG_NAMES[cfg] + (" (small)" if small else ""), "N_per_gpu": int(wl.N),
            "tokens_per_gpu": int(lens.sum()), "blocks_per_gpu": int((lens // 16).sum()),
            "table_slots": int(cache.t_keys.shape[0]), "radix_nodes": int(cache.radix.V) if cache.radix is not None else 0,
            "block_size": 16, "parallelism": "independent batches per GPU, no collective" if world > 1 else "one GPU",
            "l2": "256 MB buffer written between timed steps"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    wl, cache = cpu_inputs(args.config, args.seed, args.small)
    # the same sample rule as the cpu_baseline leg (size_sample); the per-pass budget shrinks with the
    # number of passes so that warm-up + timed steps end within a few minutes
    budget = min(args.cpu_seconds, 150.0 / max(args.steps + args.warmup, 1))
    n = size_sample(wl, cache, budget)
    for _ in range(args.warmup):
        oracle_pass(wl, cache, n)
    t = 0.0
    for _ in range(args.steps):
        t += oracle_pass(wl, cache, n)[0]
    value = n * args.steps / t
    sample = "each step = the oracle on " + sample_text(n, wl.N)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0,
            "ranks": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64/int32",
            "data": "synthetic", "gpu_launches": 0,
            "config": config_dict(args.config, args.small, wl, cache, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------
# steady-state cycle: the queue is resident, a cycle brings M arrivals
# ------------------------------------------------------------------------------------------
def cycle_measurement(inp, out, Ms=(32, 1000, 100000), cycles: int = 5):
    """Per cycle: H2D of the M arrivals' tokens (pinned), peek_block_hash of the arrivals only,
    peek_pending_tree_update (no rebuild), peek_lpm and peek_demand_rank over the queue, D2H of hit,
    cLPM order and demand.  The arrivals are the last M requests of the workload; the old queue's
    hashes and tree are resident from the previous cycle."""
    from paper_2607_02525_b200 import binding as B
    dev = inp.tok.device
    N = inp.N
    res = {}
    off_h = inp.off.cpu()
    bo_h = out["bo"].cpu()
    h_full, bo_full = out["h"], out["bo"].clone()
    h_hit = torch.empty(N, dtype=torch.int32).pin_memory()
    h_ord = torch.empty(N, dtype=torch.int32).pin_memory()
    h_dem = torch.empty(inp.S, dtype=torch.int32).pin_memory()
    for M in Ms:
        if M >= N:
            continue
        m = M
        while m < min(N - 1, M + 64) and int(off_h[N - m]) % 4:  # the arrivals' tokens start 16-byte aligned
            m += 1
        if int(off_h[N - m]) % 4:
            continue
        t0, b0 = int(off_h[N - m]), int(bo_h[N - m])
        tail = inp.tok[t0:]
        host_tok = tail.cpu().pin_memory()
        off_arr = (inp.off[N - m:] - t0).contiguous()
        nb_arr = int(bo_h[N]) - b0
        old = B.peek_pending_tree(h_full[:b0] if b0 else h_full[:0], bo_full[: N - m + 1].contiguous(), signals=False)
        remap = torch.arange(N - m, dtype=torch.int32, device=dev)
        bo_arr = torch.empty(m + 1, dtype=torch.int64, device=dev)
        h_arr = h_full[b0:] if nb_arr else torch.empty(1, dtype=torch.uint64, device=dev)

        def cycle():
            tail.copy_(host_tok, non_blocking=True)
            B.peek_block_hash(tail, off_arr, nb_arr, blk_off=bo_arr, hashes=h_arr)  # hashes land in the queue's array
            bo_full[N - m:] = bo_arr + b0
            tree = B.peek_pending_tree_update(h_full, bo_full, m, old, remap)
            hr, hh = B.peek_lpm(inp.tok, inp.off, h_full, bo_full, radix=inp.radix, t_keys=inp.keys, tree=tree)
            hit = hr if hr is not None else hh
            dem, order = B.peek_demand_rank(h_full, bo_full, tree=tree, t_keys=inp.keys, hit=hit,
                                            cluster_size=tree.cluster_size, arrival=inp.arrival)
            h_hit.copy_(hit, non_blocking=True)
            h_ord.copy_(order, non_blocking=True)
            h_dem.copy_(dem, non_blocking=True)
            return tree, hit
        tree, hit = cycle()
        torch.cuda.synchronize()
        same = bool(torch.equal(tree.order, out["tree"].order) and torch.equal(tree.lcp, out["tree"].lcp)
                    and torch.equal(hit, out["hit"]))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(cycles):
            cycle()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / cycles
        res[str(M)] = {"arrivals": m, "ms_per_cycle": ms, "queries_per_s": N / (ms * 1e-3),
                       "h2d_bytes_per_cycle": int(host_tok.numel() * 4),
                       "d2h_bytes_per_cycle": int(N * 8 + inp.S * 4),
                       "equals_rebuild": same}
    return res


# ------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------
def run_peek(args):
    import torch.distributed as dist
    from paper_2607_02525_b200 import binding as B
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl peek needs a CUDA device (there is no CPU path)")
    if local >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d has no GPU (%d visible): --gpus must not exceed the GPUs of the node"
                         % (local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()  # fail loudly now if libpeek.so is missing

    # each rank owns an independent batch (its own queue and cache replica): weak scaling, no
    # data-path collective
    inp = build_inputs(args.config, rank_seed(args.seed, rank), args.small, dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    peak, peak_src = measured_peak()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        out = step(inp)
    torch.cuda.synchronize()
    launches0 = B.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    ms_list, prof, out = time_steps(inp, args.steps, flush)  # L2 flushed between timed steps, outside the event pairs
    barrier()
    t_ms = float(sum(ms_list))
    launches = (B.launch_count() - launches0) // max(args.steps, 1)
    # keep the same load running ~1.5 s more so the clock sampler sees it (not timed)
    t_end = time.time() + 1.5
    while time.time() < t_end:
        step(inp)
        torch.cuda.synchronize()
    clocks = sampler.stop()
    rank_ms = t_ms
    t_ms = max_over_ranks(t_ms, dev, world)
    all_clocks = [clocks]
    if world > 1:
        gathered = [None] * world
        dist.all_gather_object(gathered, {"rank": rank, "ms_per_step": rank_ms / args.steps, "clocks": clocks})
        all_clocks = gathered
    sum_hit = int(out["hit"].long().sum().item())

    # end to end: host buffers in, results out, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        h_tok = inp.tok.cpu().pin_memory()
        h_off = inp.off.cpu().pin_memory()
        d_tok = torch.empty_like(inp.tok)
        d_off = torch.empty_like(inp.off)
        h_hit = torch.empty(inp.N, dtype=torch.int32).pin_memory()
        h_ord = torch.empty(inp.N, dtype=torch.int32).pin_memory()
        h_dem = torch.empty(inp.S, dtype=torch.int32).pin_memory()

        def e2e_step():
            d_tok.copy_(h_tok, non_blocking=True)
            d_off.copy_(h_off, non_blocking=True)
            o = step(inp, d_tok, d_off)
            h_hit.copy_(o["hit"], non_blocking=True)
            h_ord.copy_(o["clpm"], non_blocking=True)
            h_dem.copy_(o["demand"], non_blocking=True)
        e2e_step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.e2e_steps):
            e2e_step()
        e1.record()
        barrier()
        te_ms = max_over_ranks(e0.elapsed_time(e1), dev, world)
        e2e = {"value": job_throughput(inp.N, world, args.e2e_steps, te_ms), "unit": UNIT,
               "h2d_bytes_per_step": int(h_tok.numel() * 4 + h_off.numel() * 8),
               "d2h_bytes_per_step": int(inp.N * 8 + inp.S * 4), "steps": args.e2e_steps,
               "ms_per_step": te_ms / args.e2e_steps,
               "what": "every step re-uploads and re-hashes the whole queue (PCIe bound); the cycle the method "
                       "runs - arrivals only - is under `cycle`"}
        del h_tok, d_tok

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # roofline of the dominant kernel group
    calls = calls_table(inp, prof, out, args.steps, t_ms)
    ceil = gather_ceiling(inp, dev)
    if "hbm" in ceil:
        for slot in ("lpm.radix_walk", "lpm.hash_probe", "lpm.dual_walk", "demand.count"):
            if slot in calls and "alg_GBps" in calls[slot]:
                calls[slot]["frac_of_random_sector_ceiling"] = calls[slot]["alg_GBps"] / ceil["hbm"]["GBps"]
    dom = max(calls, key=lambda s: calls[s]["ms_per_step"])
    dom_ms = prof[dom][0] / max(prof[dom][1], 1)
    dom_bytes = calls[dom].get("alg_bytes", 0)
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
    cfgd = config_dict(args.config, args.small, inp.wl, inp.cache, world)
    cfgd["l2"] += "; inputs %.1f GB" % (inp.T * 4 / 1e9)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src, "traffic": ncu_traffic(cfgd["workload"], dom),
                "traffic_source": "profiles/ncu_traffic.csv, matched on the kernel source's sha (%s)" % kernel_source_sha(dom),
                "alg_bytes_per_launch": dom_bytes, "ms_per_launch": dom_ms}
    pair = pair_summary(calls, peak)
    pair["dram_bytes_ncu"] = {s: ncu_traffic(cfgd["workload"], s) for s in pair["kernels"]}
    line = {"metric": METRIC, "value": job_throughput(inp.N, world, args.steps, t_ms), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": t_ms / args.steps,
            "ms_per_step_median": float(np.median(ms_list)), "ms_per_step_best": float(min(ms_list)),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64/int32",
            "data": "synthetic", "config": cfgd,
            "tokens_matched_per_s": world * sum_hit * args.steps / (t_ms * 1e-3),
            "gpu_launches": int(launches), "clocks": clocks, "ranks": all_clocks if world > 1 else None,
            "e2e": e2e, "roofline": roofline, "north_star_pair": pair, "calls": calls,
            "random_sector_gather_ceiling": ceil, "next_rows": next_rows_timing(inp, out),
            "work_counters": work_counters(inp, out)}
    if world == 1 and not args.no_cycle:
        line["cycle"] = cycle_measurement(inp, out)
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        n = size_sample(inp.wl, inp.cache, args.cpu_seconds)
        dt, orc = oracle_pass(inp.wl, inp.cache, n, keep=True)
        line["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                                "sample": sample_text(n, inp.N) + ", same cache, one pass of "
                                          "hash+tree+lpm(radix,hash)+demand+rank in %.2f s" % dt}
        line["parity_in_run"] = parity_in_run(inp, n, orc, out, True)
        del orc
    if world == 1 and not args.no_per_config and not args.small:
        # the other configs of BASELINE.json, timed in the same run: median and best of
        # 20 passes, flushed; configs 1-2 fit in L2 and are also timed warm
        per = {}
        main_inp = inp
        del inp, out
        for cfg in (1, 2, 3, 4, 5):
            if cfg == args.config:
                ci = main_inp
            else:
                ci = build_inputs(cfg, args.seed, False, dev)
            per[CONFIG_NAMES[cfg]] = config_summary(ci, 20, flush, peak, warm_too=cfg in (1, 2))
            if ci is not main_inp:
                del ci
                torch.cuda.empty_cache()
        line["per_config"] = per
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(respawn_under_torchrun(args))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_peek(args)


if __name__ == "__main__":
    main()
