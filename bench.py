#!/usr/bin/env python
"""bench.py — decode-attention µs/step and achieved HBM GB/s (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4] [--impl reference]

A "step" is one pass of the whole hot path (ONE launch of the split-KV
kernel, whose last-arriving CTA per cut segment runs the LSE combine) over one synthetic decode batch.  The default workload is BASELINE.json configs[1] (C2: batch 1,
64q/8kv heads, D 128, 32 768-token context, page_size 16, pages permuted in a 4 096-page pool).

What the ONE JSON line on stdout holds (rank 0):
  value / ms_per_step  whole-job GB/s = algorithmic KV+Q bytes of all ranks / max-over-ranks device
                       time of EXACTLY K steps, inputs resident in HBM, CUDA events on the launch stream
  roofline             the dominant (only) kernel: algorithmic bytes per launch / its average launch
                       duration over the timed region, against MEASURED_PEAKS.json's hbm_gbs; the un-fused
                       split phase timed alone is reported beside it as `split_only_us`
  e2e                  the same metric through comem_decode_step_host: every step brings q and the new
                       (k, v) rows from pinned host memory, appends, attends, and lands out in host memory
                       (the kernels move those bytes themselves over the host link), host-synchronous
  cpu_baseline         the fp64 oracle (oracle/, test infrastructure) on this box's host cores
  parity               GPU vs oracle on the bench's own inputs (max-abs / mean-abs / rel-l2)

L2-cold rule: C2's KV (128 MiB) is about one L2 (126 MB), so steps rotate over R = 8 disjoint pools
(2 GiB of K+V); C3/C4 read 4.8 / 8.6 GB per step, nothing survives between steps.

`--impl reference`: this tier has no reference implementation; the arm times the oracle, as it
stands, on a bounded sample of the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "decode_attn_achieved_hbm_gbs"
UNIT = "GB/s"
FALLBACK_PEAK_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback
L2_BYTES_NOMINAL = 126e6

TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")
# COMEM_LAUNCH_* bits the decode workloads are launched with unless --launch-flags says otherwise
DEFAULT_LAUNCH_FLAGS = 7  # KV_PREFIX_IMMUTABLE | SPLIT_COMBINE | Q_STABLE: nothing in the timed loops writes the cache prefix or q


def kernel_source_sha() -> str:
    """sha256 over the kernel sources a traffic capture belongs to (the attention kernels and what they include)."""
    import hashlib

    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2605_30842_b200", "csrc")
    for f in ("decode_split.cu", "merge.cuh", "schedule.cuh", "ptx.cuh", "decode_params.cuh", "prefill_attn.cu", "tcgen05.cuh",
              "decode_fp8_tc.cu"):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the workload's kernel from the committed
    `ncu --set full` capture recorded in profiles/ncu_traffic.json -- or None when that capture was taken on other
    kernel sources than the ones in the tree (a stale number is worse than none)."""
    try:
        with open(TRAFFIC_FILE) as fh:
            t = json.load(fh)
        if t.get("kernel_source_sha") != kernel_source_sha():
            return None
        return t["traffic_bytes_per_launch"].get(key)
    except Exception:  # noqa: BLE001
        return None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8192)
    ap.add_argument("--warmup", type=int, default=64)
    ap.add_argument("--workload", default="c2", choices=["c2", "c3", "c4", "c5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--affine", action="store_true",
                    help="P:L184 check: sweep the context at batch 16 and fit t = a + b*L (extra, not the bench line)")
    ap.add_argument("--window", type=int, default=0,
                    help="extra: time comem_decode_attn_window_async on the C4 batch with this sliding window")
    ap.add_argument("--sinks", type=int, default=64, help="attention-sink tokens for --window")
    ap.add_argument("--kv-fp8", action="store_true",
                    help="extra: time comem_decode_attn_fp8_async (E4M3 cache + page scales) on --workload c2|c3|c4")
    ap.add_argument("--kv-layout", default="nhd", choices=["nhd", "hnd"],
                    help="for --kv-fp8: pools [P, page, Hkv, D] (nhd) or [P, Hkv, page, D] (hnd)")
    ap.add_argument("--pipeline", type=int, default=0, metavar="K",
                    help="extra: drive 64 agent steps of the k-step-off pipeline (Algorithm 1) from comem_kstep_plan "
                         "and check eq. 5 against the measured decode-attention times")
    ap.add_argument("--offload", action="store_true",
                    help="extra: decode attention over the two-tier (HBM + pinned host) cache; prints its own line")
    ap.add_argument("--prefill", action="store_true",
                    help="extra: time comem_prefill_attn_async (paged causal prefill, tcgen05) and print its own line")
    ap.add_argument("--primary-only", action="store_true",
                    help="default run without the C3 / C4 / C5 / prefill / read-ceiling blocks of the JSON line")
    ap.add_argument("--no-graph", action="store_true", help="launch every step from the host")
    ap.add_argument("--launch-flags", type=int, default=None,
                    help="COMEM_LAUNCH_* bits for the decode calls (default: KV_PREFIX_IMMUTABLE | SPLIT_COMBINE, see DESIGN.md)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-budget-s", type=float, default=120.0,
                    help="--impl reference: wall-clock budget for the whole run")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------
def workload_desc(name: str) -> dict:
    if name == "c2":
        return {"workload": "C2 agent decode: batch 1, 64q/8kv, D128, ctx 32768, page 16, 4096-page pool",
                "batch": 1, "num_q_heads": 64, "num_kv_heads": 8, "head_dim": 128, "page_size": 16,
                "context": 32768}
    if name == "c3":
        return {"workload": "C3 agent decode: batch 32, 64q/8kv, D128, ctx U[8192,65536], page 16",
                "batch": 32, "num_q_heads": 64, "num_kv_heads": 8, "head_dim": 128, "page_size": 16,
                "context": "U[8192,65536] seed 1003"}
    return {"workload": "C4 memory-model decode: batch 16, 32q/8kv, D128, ctx 131072, page 32, 1% peaked keys",
            "batch": 16, "num_q_heads": 32, "num_kv_heads": 8, "head_dim": 128, "page_size": 32,
            "context": 131072}


def make_pools(name: str, device, rank: int, spare_tokens: int):
    """The rotating set of decode batches for one rank (seeds differ per rank and per pool)."""
    from paper_2605_30842_b200 import workloads as W

    if name == "c2":
        pools = []
        for i in range(8):
            pools.append(W.make_batch([32768], 64, 8, 128, 16, 1002 + i + 100 * rank, device, k_scale=0.5,
                                      num_pages=4096,
                                      max_pages_per_seq=W.pages_needed(32768 + spare_tokens, 16),
                                      spare_tokens=spare_tokens, name="C2-agent-1x32K"))
        return pools
    if name == "c3":
        return [W.config3_agent_ragged(device, spare_tokens=spare_tokens)]
    return [W.make_batch([131072] * 16, 32, 8, 128, 32, 1004 + 100 * rank, device,
                         num_pages=16 * W.pages_needed(131072 + spare_tokens, 32) + 4096,
                         max_pages_per_seq=max(4096, W.pages_needed(131072 + spare_tokens, 32)),
                         spare_tokens=spare_tokens, peaked_frac=0.01, peaked_offset=4.0,
                         name="C4-memory-16x128K")]


# ---------------------------------------------------------------------------------------------
# clocks (sampled DURING the timed regions)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """Polls NVML every few ms from a thread: SM clock and clock-event (throttle) reasons."""

    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, uuid: str, index: int):
        self.samples, self.reasons, self.active = [], set(), False
        self.warm_samples, self.warm = [], False   # `warm`: the run-up under the same load as the timed region
        self.max_mhz, self.err = None, None
        self._stop = threading.Event()
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid).encode())
            except Exception:  # noqa: BLE001
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self._reasons_fn = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        except Exception as e:  # noqa: BLE001
            self.nv, self.err = None, repr(e)
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set():
            if (self.active or self.warm) and self.nv is not None:
                try:
                    mhz = int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                    r = int(self._reasons_fn(self.h))
                    (self.samples if self.active else self.warm_samples).append(mhz)
                    for bit, nm in self.REASONS.items():
                        if r & bit:
                            self.reasons.add(nm)
                except Exception as e:  # noqa: BLE001
                    self.err = repr(e)
            # a timed region may last half a millisecond: wake often enough to see its start, poll fast inside it
            time.sleep(0.00005 if self.active else 0.0002)

    def start(self):
        self.t.start()

    def stop(self):
        self._stop.set()
        self.t.join(timeout=1.0)

    def reset(self):
        self.samples, self.warm_samples, self.reasons = [], [], set()

    def summary(self) -> dict:
        s = sorted(self.samples)
        w = sorted(self.warm_samples)
        use = s if s else w
        out = {"sm_mhz": (use[len(use) // 2] if use else None), "sm_max_mhz": self.max_mhz,
               "reasons": sorted(self.reasons), "samples": len(s), "samples_run_up_same_load": len(w)}
        if self.err:
            out["error"] = self.err
        return out


# ---------------------------------------------------------------------------------------------
# the timed loops
# ---------------------------------------------------------------------------------------------
def timed_steps(torch, comem, replicas, pools, outs, ws, stream, steps, warmup, phases, use_graph, sampler,
                device, flags=0):
    """`warmup` untimed steps, then EXACTLY `steps` steps on `stream`, bracketed by barrier +
    synchronize on both sides; CUDA events on that stream.  With graphs (the default) every timed step is
    replayed from a CUDA graph whatever `steps` is: steps = a * C + r runs as a replays of a C-step graph and one
    replay of an r-step graph, C = min(steps, 1024) (the pools rotate inside the graph).  Returns this rank's milliseconds."""
    R = len(pools)

    def enqueue(first, n):
        for i in range(first, first + n):
            b = pools[i % R]
            comem.comem_decode_attn_phases_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                                 b.softmax_scale, outs[i % R], ws, stream=stream, phases=phases,
                                                 flags=flags)

    def capture(first, n):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            enqueue(first, n)
        return g

    with torch.cuda.stream(stream):
        enqueue(0, max(warmup, 3))
        stream.synchronize()
        # one graph for the whole timed region when it is short (no graph-launch boundary inside it: consecutive
        # steps overlap through programmatic launch only inside a graph); 1 024-step graphs for long runs
        chunk = min(steps, 1024)
        a, r = divmod(steps, chunk) if use_graph else (0, 0)
        g_full = capture(0, chunk) if a else None
        g_rest = capture(a * chunk, r) if r else None
        # the run-up: the same graphs at the same rate as the timed region, for >= 30 ms, so that the clock sampler
        # (an NVML query takes about a millisecond) has a record of the SM clock under this very load even when the
        # timed region itself lasts half a millisecond
        for g in (g_full, g_rest):
            if g is not None:
                r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                r0.record(stream)
                g.replay()
                r1.record(stream)
                stream.synchronize()
                n_run = max(3, min(2000, int(30.0 / max(r0.elapsed_time(r1), 1e-3)) + 1)) if use_graph else 3
                sampler.warm = True
                for _ in range(n_run):
                    g.replay()
                stream.synchronize()
                sampler.warm = False
        stream.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        replicas.barrier()
        torch.cuda.synchronize(device)
        sampler.warm = False
        sampler.active = True
        e0.record(stream)
        if use_graph:
            for _ in range(a):
                g_full.replay()
            if g_rest is not None:
                g_rest.replay()
        else:
            enqueue(0, steps)
        e1.record(stream)
        torch.cuda.synchronize(device)
        sampler.active = False
        replicas.barrier()
    return e0.elapsed_time(e1)


def step_distribution(torch, comem, pools, outs, ws, stream, n, phases):
    """Each of n single steps timed on its own with a CUDA-event pair (host launches, the stream idle
    before each step, so launch latency is inside): min / median / p95 in microseconds.  The headline
    number is the back-to-back one; this is the spread SURVEY.md §8(d) asks for."""
    R = len(pools)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    with torch.cuda.stream(stream):
        for i in range(n):
            b = pools[i % R]
            stream.synchronize()
            ev[i][0].record(stream)
            comem.comem_decode_attn_phases_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                                 b.softmax_scale, outs[i % R], ws, stream=stream, phases=phases)
            ev[i][1].record(stream)
        stream.synchronize()
    us = sorted(a.elapsed_time(b) * 1e3 for a, b in ev)
    return {"n": n, "min": us[0], "median": us[n // 2], "p95": us[min(n - 1, int(0.95 * n))]}


def timed_e2e(torch, comem, replicas, pools, ws, stream, steps, warmup, sampler, device, seed_base):
    """End to end through comem_decode_step_host: per step H2D(q, new k, new v) from pinned host
    memory -> append -> attention -> D2H(out), host-synchronous.  Returns (ms, bytes, h2d, d2h)."""
    from paper_2605_30842_b200 import workloads as W

    R = len(pools)
    nrows = 4  # distinct pre-generated host rows per pool, cycled (no RNG in the timed loop)
    host = []
    for i, b in enumerate(pools):
        rows = []
        for j in range(nrows):
            q, nk, nv = W.decode_step_rows(b, j, seed_base + 16 * i)
            rows.append(tuple(t.cpu().pin_memory() for t in (q, nk, nv)))
        host.append(rows)
    out_h = [torch.empty(tuple(b.q.shape), dtype=torch.bfloat16).pin_memory() for b in pools]
    per_tok = [b.batch * b.num_kv_heads * b.head_dim * 2 * 2 for b in pools]
    base = [b.algorithmic_bytes() for b in pools]
    visits = [0] * R
    h2d = sum(t.numel() * 2 for t in host[0][0])
    d2h = out_h[0].numel() * 2

    # the binding's pre-marshalled form of the call (comem.DecodeStepHost: same C entry point, arguments converted once
    # per (pool, host row set) instead of per step)
    bound = [[comem.DecodeStepHost(*host[p][j], pools[p].k_pages, pools[p].v_pages, pools[p].block_table,
                                   pools[p].seq_lens, pools[p].softmax_scale, out_h[p], ws, stream=stream)
              for j in range(nrows)] for p in range(R)]

    def step(i):
        p = i % R
        bound[p][visits[p] % nrows]()
        visits[p] += 1
        return base[p] + visits[p] * per_tok[p]  # context grew by one token per earlier visit

    for i in range(max(warmup, 3)):
        step(i)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier()
    torch.cuda.synchronize(device)
    sampler.active = True
    t0 = time.perf_counter()
    e0.record(stream)
    nbytes = 0
    for i in range(steps):
        nbytes += step(max(warmup, 3) + i)
    e1.record(stream)
    torch.cuda.synchronize(device)
    wall_ms = (time.perf_counter() - t0) * 1e3
    sampler.active = False
    replicas.barrier()
    return max(e0.elapsed_time(e1), wall_ms), nbytes, h2d, d2h


# ---------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): the only places bench.py runs oracle/
# ---------------------------------------------------------------------------------------------
def oracle_inputs_cpu(batch, seqs):
    """Gather the pages of sequences `seqs` into a compact CPU pool (pure data movement)."""
    import torch
    from paper_2605_30842_b200 import workloads as W

    ps = batch.page_size
    lens = batch.seq_lens.cpu()
    ids, off = [], 0
    maxp = max(1, max(W.pages_needed(int(lens[b]), ps) for b in seqs))
    bt = torch.zeros((len(seqs), maxp), dtype=torch.int32)
    for i, b in enumerate(seqs):
        n = W.pages_needed(int(lens[b]), ps)
        ids.append(batch.block_table[b, :n].to(torch.int64))
        bt[i, :n] = torch.arange(off, off + n, dtype=torch.int32)
        off += n
    ids = torch.cat(ids)
    sel = torch.tensor(list(seqs), dtype=torch.int64)
    return (batch.q.cpu()[sel].contiguous(), batch.k_pages[ids.to(batch.k_pages.device)].cpu(),
            batch.v_pages[ids.to(batch.v_pages.device)].cpu(), bt, lens[sel].contiguous())


def cpu_baseline_and_parity(batch, gpu_out, budget_s=20.0):
    """Time the oracle on a bounded sample of `batch` (all host cores) and compare the GPU's output
    on the same rows.  Sample: whole sequences, first-come, until ~budget_s of CPU work."""
    import numpy as np
    import oracle

    oracle.build()
    cores = oracle.max_threads()
    lens = [int(x) for x in batch.seq_lens.cpu()]
    hq, g = batch.num_q_heads, batch.num_q_heads // batch.num_kv_heads
    # calibrate on one row of sequence 0
    q, kp, vp, bt, sl = oracle_inputs_cpu(batch, [0])
    t0 = time.perf_counter()
    oracle.decode_attn(q, kp, vp, bt, sl, batch.softmax_scale, pairs=[(0, 0)], num_threads=1)
    row_s_per_tok = (time.perf_counter() - t0) / max(1, lens[0])
    seqs, est = [], 0.0
    for b, l in enumerate(lens):
        cost = row_s_per_tok * l * hq / max(1, cores) * 1.5
        if seqs and est + cost > budget_s:
            break
        seqs.append(b)
        est += cost
    if seqs != [0]:
        q, kp, vp, bt, sl = oracle_inputs_cpu(batch, seqs)
    reps = 3 if est * 3 <= budget_s else 1
    best = float("inf")
    for _ in range(reps):
        t0 = time.perf_counter()
        ref, _ = oracle.decode_attn(q, kp, vp, bt, sl, batch.softmax_scale)
        best = min(best, time.perf_counter() - t0)
    toks = sum(lens[b] for b in seqs)
    nbytes = toks * batch.num_kv_heads * batch.head_dim * 4 + len(seqs) * hq * batch.head_dim * 2
    got = gpu_out[seqs].double().cpu().numpy()
    d = np.abs(got - ref)
    parity = {"rows": len(seqs) * hq, "max_abs": float(d.max()), "mean_abs": float(d.mean()),
              "rel_l2": float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300)),
              "tol": {"max_abs": 2e-2, "mean_abs": 2e-3, "rel_l2": 5e-3}}
    parity["ok"] = bool(parity["max_abs"] <= 2e-2 and parity["mean_abs"] <= 2e-3 and parity["rel_l2"] <= 5e-3)
    # one thread, on one query head of the first sampled sequence (scaled to bytes of KV consumed)
    t0 = time.perf_counter()
    oracle.decode_attn(q, kp, vp, bt, sl, batch.softmax_scale, pairs=[(0, 0)], num_threads=1)
    one = time.perf_counter() - t0
    one_gbs = lens[seqs[0]] * batch.head_dim * 4 / g / one / 1e9   # a head reads 1/G of its kv head's K+V
    base = {"value": nbytes / best / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "single_thread_value": one_gbs,
            "sample": f"{len(seqs)} of {len(lens)} sequences, all {hq} query heads, full context "
                      f"({toks} tokens), best of {reps}; {best:.3f} s per pass",
            "seconds": best}
    return base, parity


def run_reference(args, rank: int) -> int:
    """--impl reference: the oracle, as it stands, on host cores, K steps of a bounded sample of the
    same workload (rank 0 only; other ranks exit 0 without work)."""
    if rank != 0:
        return 0
    import numpy as np  # noqa: F401
    import oracle
    from paper_2605_30842_b200 import workloads as W

    oracle.build()
    cores = oracle.max_threads()
    if args.workload == "c5":
        args.workload = "c3"  # C5's agent batch is C3; the oracle arm has no streams to overlap
    desc = workload_desc(args.workload)
    # The sample is a prefix of sequence 0's context, all query heads: T tokens chosen from a
    # calibration pass so that (warmup + steps) passes fit the budget.
    hq, hkv, d, ps = desc["num_q_heads"], desc["num_kv_heads"], desc["head_dim"], desc["page_size"]
    full_ctx = {"c2": 32768, "c3": 36864, "c4": 131072}[args.workload]
    calib = W.make_batch([4096], hq, hkv, d, ps, 4242, "cpu", k_scale=0.5 if args.workload == "c2" else 1.0)
    oracle.decode_attn(calib.q, calib.k_pages, calib.v_pages, calib.block_table, calib.seq_lens, calib.softmax_scale)
    t0 = time.perf_counter()
    oracle.decode_attn(calib.q, calib.k_pages, calib.v_pages, calib.block_table, calib.seq_lens, calib.softmax_scale)
    s_per_tok = (time.perf_counter() - t0) / 4096
    n_pass = args.steps + max(args.warmup, 1)
    T = int(min(full_ctx, max(ps, args.ref_budget_s / n_pass / s_per_tok / 1.3)))
    T = max(ps, T // ps * ps)
    b = W.make_batch([T], hq, hkv, d, ps, 1002, "cpu", k_scale=0.5 if args.workload == "c2" else 1.0,
                     name=f"{args.workload}-prefix-{T}")
    run = lambda: oracle.decode_attn(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale)  # noqa: E731
    for _ in range(max(args.warmup, 1)):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    sec = time.perf_counter() - t0
    nbytes = b.algorithmic_bytes()
    value = nbytes * args.steps / sec / 1e9
    cfg = dict(desc)
    cfg["l2"] = "n/a (host)"
    sample = (f"each step = all {hq} query heads over the first {T} of {full_ctx} tokens of one sequence "
              f"({nbytes} algorithmic bytes), fp64 oracle, {cores} OpenMP threads")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": cfg, "gpu_launches": 0,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


def measure_c5(args, torch, comem, device, reps=None) -> dict:
    """BASELINE.json configs[4]: the agent batch (C3) and the memory-model batch on two CUDA streams,
    64 successive decode steps each (append one token per sequence, then attend).  Each stream alone, both
    overlapped with full grids (time sharing), both overlapped under the library's SM-partition policy
    (comem_sm_partition + per-call launch options), and the aggregate GB/s over the overlapped window."""
    from paper_2605_30842_b200 import workloads as W

    n_steps = 64
    agent = W.config3_agent_ragged(device, spare_tokens=n_steps)
    memory = W.config5_memory_ragged(device, spare_tokens=n_steps)
    sa, sm = torch.cuda.Stream(device), torch.cuda.Stream(device)
    jobs = []
    for b, st, seed in ((agent, sa, 1005_000), (memory, sm, 1005_500)):
        jobs.append({"b": b, "stream": st, "len0": b.seq_lens.clone(),
                     "rows": [W.decode_step_rows(b, i, seed) for i in range(n_steps)],
                     "out": torch.empty_like(b.q),
                     "ws": comem.alloc_workspace(b.q, b.k_pages, b.block_table, stream=st)})
    torch.cuda.synchronize(device)

    def nbytes(j):  # algorithmic bytes of the 64 steps: the context grows by one token per step
        b = j["b"]
        l0 = int(j["len0"].sum().item())
        per_tok = b.num_kv_heads * b.head_dim * 4
        return sum((l0 + (i + 1) * b.batch) * per_tok + b.batch * b.num_q_heads * b.head_dim * 2
                   for i in range(n_steps))

    by_a, by_m = nbytes(jobs[0]), nbytes(jobs[1])
    sms = comem.comem_grid_ctas(128)
    part = comem.comem_sm_partition(by_a, by_m, sms)

    def enqueue(j, i, grid=None):
        b, st = j["b"], j["stream"]
        q, nk, nv = j["rows"][i]
        comem.comem_kv_append_async(b.k_pages, b.v_pages, b.block_table, b.seq_lens, nk, nv, stream=st)
        comem.comem_decode_attn_async(q, b.k_pages, b.v_pages, b.block_table, b.seq_lens, b.softmax_scale,
                                      j["out"], j["ws"], stream=st, grid_ctas=grid,
                                      programmatic_launch=None if grid is None else False)

    def run(which, grids=None):
        for j in jobs:
            j["b"].seq_lens.copy_(j["len0"])
        torch.cuda.synchronize(device)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in jobs]
        t0 = torch.cuda.Event(enable_timing=True)
        t0.record(torch.cuda.current_stream(device))
        for k in which:
            jobs[k]["stream"].wait_event(t0)
            ev[k][0].record(jobs[k]["stream"])
        for i in range(n_steps):
            for k in which:
                enqueue(jobs[k], i, None if grids is None else grids[k])
        for k in which:
            ev[k][1].record(jobs[k]["stream"])
        torch.cuda.synchronize(device)
        return {k: (t0.elapsed_time(ev[k][1]), ev[k][0].elapsed_time(ev[k][1])) for k in which}

    run([0, 1])  # warm-up
    if reps is None:
        reps = max(1, min(5, args.steps // n_steps if args.steps >= n_steps else 1))
    alone_a = min(run([0])[0][1] for _ in range(reps))
    alone_m = min(run([1])[1][1] for _ in range(reps))
    both = [run([0, 1]) for _ in range(reps)]
    best = min(both, key=lambda r: max(r[0][0], r[1][0]))
    window = max(best[0][0], best[1][0])
    pboth = [run([0, 1], grids=part) for _ in range(reps)]
    pbest = min(pboth, key=lambda r: max(r[0][0], r[1][0]))
    pwindow = max(pbest[0][0], pbest[1][0])
    share_a = part[0] / sms
    return {"n_steps": n_steps, "bytes_agent": by_a, "bytes_memory": by_m, "window_ms": window,
            "aggregate_gbs": (by_a + by_m) / (window * 1e-3) / 1e9,
            "agent_alone_us_per_step": alone_a / n_steps * 1e3, "memory_alone_us_per_step": alone_m / n_steps * 1e3,
            "overlapped_window_us_per_step": window / n_steps * 1e3,
            "agent_overlapped_us_per_step": best[0][1] / n_steps * 1e3,
            "memory_overlapped_us_per_step": best[1][1] / n_steps * 1e3,
            "agent_slowdown": best[0][1] / alone_a, "memory_slowdown": best[1][1] / alone_m,
            "agent_alone_gbs": by_a / (alone_a * 1e-3) / 1e9, "memory_alone_gbs": by_m / (alone_m * 1e-3) / 1e9,
            "serial_sum_us_per_step": (alone_a + alone_m) / n_steps * 1e3,
            "sm_partition": {"policy": "comem_sm_partition (proportional to bytes), per-call launch options, PDL off",
                             "agent_ctas": part[0], "memory_ctas": part[1],
                             "window_us_per_step": pwindow / n_steps * 1e3,
                             "aggregate_gbs": (by_a + by_m) / (pwindow * 1e-3) / 1e9,
                             "agent_us_per_step": pbest[0][1] / n_steps * 1e3,
                             "memory_us_per_step": pbest[1][1] / n_steps * 1e3,
                             "agent_slowdown": pbest[0][1] / alone_a, "memory_slowdown": pbest[1][1] / alone_m,
                             "agent_sm_share": share_a,
                             "agent_slowdown_bound_1_over_share": 1.0 / share_a}}


def run_c5(args) -> int:
    """--workload c5: the config-5 measurement as its own JSON line (1 GPU only)."""
    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback exists)"
    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    c5 = measure_c5(args, torch, comem, device)
    line = {"metric": METRIC, "value": c5["aggregate_gbs"], "unit": UNIT, "n_gpus": 1,
            "steps": c5["n_steps"], "warmup": c5["n_steps"], "ms_per_step": c5["window_ms"] / c5["n_steps"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": "C5 k-step-off overlap: C3 agent batch + memory batch (8 x U[65536,131072], 32q/8kv) "
                                   "on two streams, 64 append+attend steps each",
                       "l2": "cold: each step reads 4.5 + 3.0 GiB of KV >> L2", "launch": "host launches, 2 kernels per step per stream"},
            "c5": c5, "gpu_launches": 4 * c5["n_steps"]}
    print(json.dumps(line), flush=True)
    return 0


def run_affine(args) -> int:
    """SURVEY.md §8(d) affine check of eq. 5 (t = L*S/W) at the paper's batch sizes (Fig. 2, L84-92: batch 1 /
    16 / 64; section 4.4: 32 -> 256): 64q/8kv, D 128, page 16, context L from 1K up to what 16 GiB of K+V hold;
    least-squares fit t = a + b*L per batch.  batch * 4096 B / b is the streaming rate W, a the fixed cost per step
    (Fig. 2's shape: flat while a dominates, linear beyond).  One JSON line; an extra, not the driver's bench line."""
    import numpy as np
    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build
    from paper_2605_30842_b200 import workloads as W

    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    stream = torch.cuda.Stream(device)
    flags = DEFAULT_LAUNCH_FLAGS if args.launch_flags is None else args.launch_flags
    rows = []
    for B in (1, 16, 64, 128, 256):
        pts = []
        for L in (1024, 4096, 8192, 16384, 32768, 65536, 131072):
            if B * L * 4096 > (16 << 30):
                continue
            R = max(1, min(8, (1 << 30) // (B * L * 4096)))          # rotate pools while one step is < 1 GiB (L2-cold)
            pools = [W.make_batch([L] * B, 64, 8, 128, 16, 7000 + i, device) for i in range(R)]
            outs = [torch.empty_like(b.q) for b in pools]
            ws = comem.alloc_workspace(pools[0].q, pools[0].k_pages, pools[0].block_table, stream=stream)
            est_us = B * L * 4096 / 7e6 + 10
            per_graph = max(R, min(256, int(5e3 / est_us)))           # short steps need a long graph (PDL overlap)
            with torch.cuda.stream(stream):
                def enq(n):
                    for i in range(n):
                        b = pools[i % R]
                        comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                                      b.softmax_scale, outs[i % R], ws, stream=stream, flags=flags)
                enq(R)
                stream.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=stream):
                    enq(per_graph)
                for _ in range(3):
                    g.replay()
                n = max(2, int(20e3 / (est_us * per_graph)))         # ~20 ms of streaming per point
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                stream.synchronize()
                e0.record(stream)
                for _ in range(n):
                    g.replay()
                e1.record(stream)
                stream.synchronize()
            us = e0.elapsed_time(e1) / (n * per_graph) * 1e3
            pts.append((L, us, pools[0].algorithmic_bytes() / us / 1e3))
            del pools, outs, ws, g
            torch.cuda.empty_cache()
        Ls, ts = np.array([p[0] for p in pts], float), np.array([p[1] for p in pts], float)
        b_fit, a_fit = np.polyfit(Ls, ts, 1)
        rows.append({"batch": B, "points": [{"L": int(l), "us_per_step": round(u, 2), "gbs": round(gb, 1)} for l, u, gb in pts],
                     "a_us": a_fit, "b_us_per_token": b_fit, "slope_gbs": B * 4096 / b_fit / 1e3,
                     "max_rel_residual": float(np.max(np.abs(a_fit + b_fit * Ls - ts) / ts))})
    print(json.dumps({"affine_check": "t_us = a + b * L per batch, 64q/8kv, D128, page 16 (PAPER.md eq. 5, Fig. 2)",
                      "launch_flags": flags, "batches": rows}), flush=True)
    return 0


def run_window(args) -> int:
    """Extra: the sliding-window + attention-sink variant on the C4 batch
    (16 x 131072 tokens, 32q/8kv, page 32).  Algorithmic bytes = K+V of the KEPT tokens + Q; the same
    HBM roofline applies to them.  One JSON line; not the driver's bench line."""
    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build
    from paper_2605_30842_b200 import workloads as W

    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    b = W.config4_memory_long(device)
    kept = sum(min(L, min(args.sinks, max(L - args.window, 0)) + min(args.window, L)) for L in b.seq_lens.cpu().tolist())
    nbytes = kept * b.num_kv_heads * b.head_dim * 4 + b.batch * b.num_q_heads * b.head_dim * 2
    R = max(1, min(8, (1 << 30) // max(nbytes, 1)))              # rotate q/out only: the pool is 17 GiB, L2-cold anyway
    stream = torch.cuda.Stream(device)
    out = torch.empty_like(b.q)
    ws = comem.alloc_workspace(b.q, b.k_pages, b.block_table, stream=stream)
    with torch.cuda.stream(stream):
        f = lambda: comem.comem_decode_attn_window_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,  # noqa: E731
                                                         b.softmax_scale, out, ws, args.window, args.sinks, stream=stream)
        f()
        stream.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            f()
        flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)   # > L2: written between timed steps
        n, tot = max(3, min(args.steps, 50)), 0.0
        for i in range(n + 3):
            flush.fill_(i & 0xff)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            g.replay()
            e1.record(stream)
            stream.synchronize()
            if i >= 3:
                tot += e0.elapsed_time(e1)
    us = tot / n * 1e3
    print(json.dumps({"extra": "sliding window + sinks on the C4 batch", "window": args.window, "sinks": args.sinks,
                      "kept_tokens": kept, "algorithmic_bytes_per_step": nbytes, "us_per_step": us,
                      "value": nbytes / us / 1e3, "unit": UNIT, "l2": "flushed (512 MiB written) before every timed step",
                      "full_attention_bytes": b.algorithmic_bytes()}), flush=True)
    return 0


def run_offload(args) -> int:
    """Extra: decode attention over the two-tier cache.  The C3 agent batch
    with the coldest 0 / 5 / 10 / 25 / 50 % of every sequence's pages in pinned host memory: us/step, and the rate at
    which the host-resident bytes crossed the host link.  One JSON line; not the driver's bench line."""
    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build
    from paper_2605_30842_b200 import workloads as W

    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    b = W.config3_agent_ragged(device)
    stream = torch.cuda.Stream(device)
    rows = []
    ref_out = None
    for frac in (0.0, 0.05, 0.10, 0.25, 0.50):
        ob = W.offload_pages(b, frac, seed=11)
        bb = ob.base
        out = torch.empty_like(bb.q)
        ws = comem.alloc_workspace(bb.q, bb.k_pages, bb.block_table, stream=stream)
        with torch.cuda.stream(stream):
            f = lambda: comem.comem_decode_attn_offload_async(bb.q, bb.k_pages, bb.v_pages, ob.k_host, ob.v_host,  # noqa: E731
                                                              bb.block_table, bb.seq_lens, bb.softmax_scale, out, ws,
                                                              stream=stream)
            for _ in range(2):
                f()
            stream.synchronize()
            n = max(3, min(args.steps, 10))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(n):
                f()
            e1.record(stream)
            stream.synchronize()
        us = e0.elapsed_time(e1) / n * 1e3
        if ref_out is None:
            ref_out = out.clone()
        same = bool(torch.equal(out.view(torch.int16), ref_out.view(torch.int16)))
        rows.append({"host_fraction": frac, "host_bytes_per_step": ob.host_bytes(), "us_per_step": us,
                     "host_link_gbs": (ob.host_bytes() / us / 1e3) if ob.host_bytes() else None,
                     "total_gbs": b.algorithmic_bytes() / us / 1e3, "bits_equal_all_hbm": same})
        del ob, bb, out, ws
    print(json.dumps({"extra": "two-tier cache (HBM + pinned host memory), C3 agent batch, coldest pages offloaded",
                      "algorithmic_bytes_per_step": b.algorithmic_bytes(), "rows": rows,
                      "note": "host-resident tiles are TMA-loaded over the host link straight into shared memory, once per step"}),
          flush=True)
    return 0


def fp8_parity(fb, gpu_out, seq: int = 0):
    """Oracle (oracle.decode_attn_fp8, all host cores) on ONE whole sequence of the FP8 batch, all its query heads,
    from the same bytes and scales; returns (parity block, oracle seconds)."""
    import numpy as np
    import torch
    import oracle

    oracle.build()
    ps = fb.page_size
    n = (int(fb.seq_lens[seq]) + ps - 1) // ps
    ids = fb.block_table[seq, :n].long()
    t0 = time.perf_counter()
    ref, _ = oracle.decode_attn_fp8(fb.q[seq:seq + 1].cpu(), fb.k_pages[ids].cpu(), fb.v_pages[ids].cpu(),
                                    fb.k_scale[ids].cpu(), fb.v_scale[ids].cpu(),
                                    torch.arange(n, dtype=torch.int32).view(1, n), fb.seq_lens[seq:seq + 1].cpu(),
                                    fb.softmax_scale, kv_layout=fb.kv_layout)
    secs = time.perf_counter() - t0
    got = gpu_out[seq:seq + 1].double().cpu().numpy()
    d = np.abs(got - ref)
    par = {"rows": fb.num_q_heads, "max_abs": float(d.max()), "mean_abs": float(d.mean()),
           "rel_l2": float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300)),
           "tol": {"max_abs": 2e-2, "mean_abs": 2e-3, "rel_l2": 5e-3}}
    par["ok"] = bool(par["max_abs"] <= 2e-2 and par["mean_abs"] <= 2e-3 and par["rel_l2"] <= 5e-3)
    return par, secs


def run_fp8(args) -> int:
    """Extra: the FP8 (E4M3 + per-page, per-kv-head scale) KV-cache variant on the
    C2 / C3 / C4 batch, quantised by the input recipe (workloads.quantize_batch_fp8).  Algorithmic bytes =
    1 B per K and V element of every token + 8 B of scales per (page, kv head) + Q; the same HBM roofline
    applies.  Steps rotate over enough pools to exceed L2 and are replayed from one CUDA graph.
    One JSON line; not the driver's bench line."""
    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build
    from paper_2605_30842_b200 import workloads as W

    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    pools = []
    for bf in make_pools(args.workload, device, 0, 64):   # 64 spare tokens per sequence: room for the e2e leg's appends
        f8 = W.quantize_batch_fp8(bf)
        del bf
        pools.append(W.to_hnd(f8) if args.kv_layout == "hnd" else f8)
        del f8
    torch.cuda.empty_cache()
    # default: the early mode + small combine for the one-sequence step (C2), the classic order for the long steps (the
    # FP8 consumers are bound by their issue slots and the early-mode instance costs them 5 % there)
    flags = ((DEFAULT_LAUNCH_FLAGS if args.workload == "c2" else 0) if args.launch_flags is None else args.launch_flags)
    nbytes = pools[0].algorithmic_bytes()
    bf16_bytes = int(pools[0].seq_lens.to(torch.int64).sum().item()) * pools[0].num_kv_heads * pools[0].head_dim * 4
    stream = torch.cuda.Stream(device)
    outs = [torch.empty_like(b.q) for b in pools]
    ws = comem.alloc_workspace(pools[0].q, pools[0].k_pages, pools[0].block_table, stream=stream,
                               kv_layout=pools[0].kv_layout)
    peaks = {"hbm_gbs": FALLBACK_PEAK_GBS}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peaks["hbm_gbs"] = float(json.load(fh)["hbm_gbs"])
    except Exception:  # noqa: BLE001
        pass
    with torch.cuda.stream(stream):
        def step(i):
            b = pools[i % len(pools)]
            comem.comem_decode_attn_fp8_async(b.q, b.k_pages, b.v_pages, b.k_scale, b.v_scale, b.block_table,
                                              b.seq_lens, b.softmax_scale, outs[i % len(pools)], ws, stream=stream,
                                              kv_layout=b.kv_layout, flags=flags)
        for i in range(len(pools)):
            step(i)
        stream.synchronize()
        est_us = nbytes / 5e6 + 8
        # (a short step needs a long graph: consecutive steps overlap through programmatic launch only inside one)
        per_graph = max(len(pools), 4, min(256, int(5e3 / est_us)))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=stream):
            for i in range(per_graph):
                step(i)
        replays = max(4, min(int(2e6 / (est_us * per_graph)), max(1, args.steps // per_graph)))
        for _ in range(3):
            g.replay()
        # burst: a short run from an idle, cool GPU (SM clock at its maximum) ...
        stream.synchronize()
        time.sleep(1.0)
        bs = ClockSampler(str(getattr(torch.cuda.get_device_properties(device), 'uuid', '')), 0)
        bs.start()
        burst_replays = max(1, min(replays, int(40e3 / (est_us * per_graph))))   # ~40 ms
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g.replay()
        stream.synchronize()
        bs.active = True
        b0.record(stream)
        for _ in range(burst_replays):
            g.replay()
        b1.record(stream)
        stream.synchronize()
        bs.active = False
        bs.stop()
        burst_us = b0.elapsed_time(b1) * 1e3 / (burst_replays * per_graph)
        # ... then the sustained run (seconds): this kernel plus HBM at full rate reaches the board's power cap
        sampler = ClockSampler(str(getattr(torch.cuda.get_device_properties(device), 'uuid', '')), 0)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        sampler.active = True
        e0.record(stream)
        for _ in range(replays):
            g.replay()
        e1.record(stream)
        stream.synchronize()
        sampler.active = False
        sampler.stop()
        # the same step launched on its own after an L2 flush (no back-to-back overlap, idle-stream launch latency inside)
        flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)
        iso = []
        for i in range(12):
            flush.fill_(i)
            i0, i1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            i0.record(stream)
            step(i)
            i1.record(stream)
            stream.synchronize()
            if i >= 2:
                iso.append(i0.elapsed_time(i1) * 1e3)
        iso.sort()
    us = e0.elapsed_time(e1) * 1e3 / (replays * per_graph)
    gbs = nbytes / us / 1e3
    with torch.cuda.stream(stream):
        step(0)
        stream.synchronize()
    parity, oracle_s = (None, None) if args.no_cpu_baseline else fp8_parity(pools[0], outs[0])
    # end to end through comem_decode_step_host_fp8: pinned host q / k / v rows in, quantising append, attention, host out
    e2e = None
    if pools[0].kv_layout in ("NHD", "HND"):
        n_e2e = 32
        rows = []
        for j in range(4):
            gq = torch.Generator(device=device)
            gq.manual_seed(4242 + j)
            b0_ = pools[0]
            rows.append(tuple(torch.randn(sh, generator=gq, device=device).to(torch.bfloat16).cpu().pin_memory()
                              for sh in (tuple(b0_.q.shape), (b0_.batch, b0_.num_kv_heads, b0_.head_dim),
                                         (b0_.batch, b0_.num_kv_heads, b0_.head_dim))))
        out_h = torch.empty(tuple(pools[0].q.shape), dtype=torch.bfloat16).pin_memory()
        lens0 = [b.seq_lens.clone() for b in pools]

        def e2e_step(i):
            b = pools[i % len(pools)]
            q, nk, nv = rows[i % 4]
            comem.comem_decode_step_host_fp8(q, nk, nv, b.k_pages, b.v_pages, b.k_scale, b.v_scale, b.block_table,
                                             b.seq_lens, b.softmax_scale, out_h, ws, stream=stream, kv_layout=b.kv_layout)
        for i in range(3):
            e2e_step(i)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(n_e2e):
            e2e_step(3 + i)
        t1 = time.perf_counter()
        for b, l0 in zip(pools, lens0):
            b.seq_lens.copy_(l0)
        e2e_us = (t1 - t0) / n_e2e * 1e6
        h2d = (rows[0][0].numel() + 2 * rows[0][1].numel()) * 2
        e2e = {"value": nbytes / e2e_us / 1e3, "unit": UNIT, "us_per_step": e2e_us, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": out_h.numel() * 2, "steps": n_e2e,
               "api": "comem_decode_step_host_fp8, pinned host buffers (host wall clock around the synchronous calls)"}
    print(json.dumps({"extra": "FP8 (E4M3 + page scales) KV cache", "config": workload_desc(args.workload), "e2e": e2e,
                      "launch_flags": flags,
                      "kv_layout": pools[0].kv_layout,
                      "pools": len(pools), "steps": replays * per_graph, "us_per_step": us,
                      "algorithmic_bytes_per_step": nbytes, "value": gbs, "unit": UNIT,
                      "frac_of_measured_peak": gbs / peaks["hbm_gbs"], "peak": peaks["hbm_gbs"],
                      "roofline": {"bound": "hbm", "kernel": "decode_fp8_tc_kernel (tcgen05 kind::f8f6f4)" if flags & 8 else "decode_split_kernel<128, 1, %d>" % (flags & 1), "achieved": gbs,
                                   "peak": peaks["hbm_gbs"], "unit": UNIT, "frac": gbs / peaks["hbm_gbs"],
                                   "us_per_launch": us,
                                   "traffic": ncu_traffic("fp8%s_%s_%s" % ("tc" if flags & 8 else "", args.workload, pools[0].kv_layout.lower()))},
                      "gpu_launches": replays * per_graph, "parity": parity, "oracle_seconds_one_sequence": oracle_s,
                      "bf16_cache_bytes_same_tokens": bf16_bytes,
                      "equivalent_bf16_gbs": bf16_bytes / us / 1e3, "clocks": sampler.summary(),
                      "burst": {"steps": burst_replays * per_graph, "us_per_step": burst_us, "value": nbytes / burst_us / 1e3,
                                "equivalent_bf16_gbs": bf16_bytes / burst_us / 1e3, "clocks": bs.summary()},
                      "isolated_step_us": {"n": len(iso), "min": iso[0], "median": iso[len(iso) // 2]},
                      "l2": "cold: steps rotate over %d pools (%.2f GiB)" % (len(pools), len(pools) * nbytes / 2 ** 30)}),
          flush=True)
    return 0


def pipeline_trajectory(torch, comem, W, device, K, T, TURN, SUMM, CONC, Y, YM):
    """The whole trajectory through the library's scheduler (comem_kstep_step_async): per agent step the prefill
    attention (cached or uncached, as Algorithm 1 says), Y decode tokens (append + decode attention), and the memory
    model's jobs on the second stream with the SM-partition policy -- once under CoMem's plan (retain-turns K) and once
    as the full-context baseline (no memory model: the plan of k > T never adopts or launches).  Eq. 6: the
    net speed-up holds iff the decode time saved per cycle exceeds the uncached prefill it costs."""
    max_ctx = T * TURN + max(Y, YM) + 16

    def build(hq, seed, cap_tokens):
        b = W.make_batch([max_ctx] * CONC, hq, 8, 128, 16, seed, device)
        qp = torch.empty((CONC * cap_tokens, hq, 128), dtype=torch.bfloat16, device=device).normal_()
        m = {"b": b, "qp": qp, "op": torch.empty_like(qp), "od": torch.empty_like(b.q),
             "nk": torch.randn((CONC, 8, 128), device=device).to(torch.bfloat16),
             "nv": torch.randn((CONC, 8, 128), device=device).to(torch.bfloat16),
             "qs": torch.zeros(CONC + 1, dtype=torch.int32, device=device),
             "ws": comem.alloc_workspace(b.q, b.k_pages, b.block_table)}
        m["model"] = comem.kstep_model(b.q, m["od"], qp, m["op"], m["nk"], m["nv"], b.k_pages, b.v_pages, b.block_table,
                                       b.seq_lens, m["qs"], m["ws"], b.softmax_scale)
        return m

    agent = build(64, 1301, SUMM + (K + 1) * TURN)   # CoMem never prefills more than summary + k + 1 turns at once
    memory = build(32, 1302, T * TURN)               # the memory model prefills the whole trajectory so far
    sa, sm = torch.cuda.Stream(device), torch.cuda.Stream(device)
    ev_done, ev_step = torch.cuda.Event(), torch.cuda.Event()
    ev_done.record(sm)
    ev_step.record(sa)
    torch.cuda.synchronize()
    out = {}
    # "comem_memory_elsewhere" is the paper's deployment (separate engines for the agent and the memory model,
    # P:L245, L310): this GPU runs the agent's side of Algorithm 1 only; "comem_colocated" also runs every memory
    # job (a full-trajectory prefill of the 32q/8kv model at the same concurrency) on this GPU's second stream.
    for name, k_plan, mem in (("comem_memory_elsewhere", K, None), ("comem_colocated", K, memory),
                              ("full_context", T + 1, None)):
        arr, events = comem.comem_kstep_plan(T, k_plan, 0)
        per_step, launches, partitioned = [], 0, 0
        t0 = torch.cuda.Event(enable_timing=True)
        t0.record(sa)
        marks = []
        for e in events:
            st = comem.comem_kstep_step_async(e, TURN, SUMM, Y, YM, agent["model"], None if mem is None else mem["model"],
                                              sa, sm, ev_done, ev_step)
            launches += st.launches
            partitioned += st.memory_in_flight
            m = torch.cuda.Event(enable_timing=True)
            m.record(sa)
            marks.append(m)
        torch.cuda.synchronize()
        prev = t0
        for m in marks:
            per_step.append(prev.elapsed_time(m))
            prev = m
        unc = [per_step[i] for i, e in enumerate(events) if e.prefill_uncached and i > 0]
        out[name] = {"agent_stream_ms": t0.elapsed_time(marks[-1]), "launches": launches,
                     "steps_with_sm_partition": partitioned, "per_step_ms": [round(x, 3) for x in per_step],
                     "uncached_prefill_steps": sum(int(e.prefill_uncached) for e in events),
                     "mean_ms_steps_with_uncached_prefill": (sum(unc) / len(unc)) if unc else None}
    out["speedup_agent_stream"] = out["full_context"]["agent_stream_ms"] / out["comem_memory_elsewhere"]["agent_stream_ms"]
    out["speedup_agent_stream_colocated"] = out["full_context"]["agent_stream_ms"] / out["comem_colocated"]["agent_stream_ms"]
    out["config"] = {"k": K, "steps": T, "turn_tokens": TURN, "summary_tokens": SUMM, "concurrency": CONC,
                     "decode_tokens_per_step": Y, "memory_decode_tokens": YM}
    return out


def run_pipeline(args) -> int:
    """Extra: the k-step-off pipeline (Algorithm 1) over 64 agent steps
    (L261), shaped like the paper's crossover benchmark (section 4.5: fixed-length turns, concurrency 32,
    k = 3; CoMem prompt bounded at a few K tokens, full-context prompt growing to ~40K).  The library's
    comem_kstep_plan says, per step, which summary is in use; the agent batch's decode attention (one layer,
    64q/8kv, D 128, page 16) is timed at the CoMem context and at the full context, L2 flushed before every
    launch; eq. 5's predicted saving (L_full - L_sum) * S / W, with S = the batch's KV bytes per token position
    and W = the slope of the measured times themselves, is compared with the measured saving.  Where a memory
    job is launched, the memory model's decode attention (32q/8kv over the full history, same concurrency) runs
    on a second stream under the agent's next steps and the agent's slowdown is reported."""
    import statistics

    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build
    from paper_2605_30842_b200 import workloads as W

    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    K, T, TURN, SUMM, CONC = args.pipeline, 64, 640, 3072, 32
    arr, events = comem.comem_kstep_plan(T, K, 0)
    ctx_comem, ctx_full, mem_in = comem.comem_kstep_context_lengths(arr, T, TURN, SUMM)
    agent = W.make_batch([T * TURN] * CONC, 64, 8, 128, 16, 1201, device, name="pipeline-agent")
    memory = W.make_batch([T * TURN] * CONC, 32, 8, 128, 16, 1202, device, name="pipeline-memory")
    sa, sb = torch.cuda.Stream(device), torch.cuda.Stream(device)
    out_a, out_m = torch.empty_like(agent.q), torch.empty_like(memory.q)
    ws_a = comem.alloc_workspace(agent.q, agent.k_pages, agent.block_table, stream=sa)
    ws_m = comem.alloc_workspace(memory.q, memory.k_pages, memory.block_table, stream=sb)
    lens_a = torch.empty(CONC, dtype=torch.int32, device=device)
    lens_m = torch.empty(CONC, dtype=torch.int32, device=device)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)
    torch.cuda.synchronize()

    def launch(b, lens, out, ws, stream):
        comem.comem_decode_attn_async(b.q, b.k_pages, b.v_pages, b.block_table, lens, b.softmax_scale, out, ws,
                                      stream=stream)

    def time_agent(ctx, reps=5):
        ts = []
        with torch.cuda.stream(sa):
            lens_a.fill_(ctx)
            for i in range(reps + 1):
                flush.fill_(i)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(sa)
                launch(agent, lens_a, out_a, ws_a, sa)
                e1.record(sa)
                sa.synchronize()
                if i:
                    ts.append(e0.elapsed_time(e1) * 1e3)
        return statistics.median(ts)

    t_comem = [time_agent(c) for c in ctx_comem]
    t_full = [time_agent(c) for c in ctx_full]
    # W from the measured times themselves: least-squares slope of t over context (both series), eq. 5's premise
    xs, ys = ctx_comem + ctx_full, t_comem + t_full
    n = len(xs)
    mx, my = sum(xs) / n, sum(ys) / n
    slope = sum((x - mx) * (y - my) for x, y in zip(xs, ys)) / sum((x - mx) ** 2 for x in xs)   # us per token
    fixed = my - slope * mx
    s_bytes = CONC * agent.num_kv_heads * agent.head_dim * 2 * 2                                  # per token position
    w_gbs = s_bytes / slope / 1e3
    rel = []
    for t in range(T):
        if ctx_full[t] - ctx_comem[t] >= 4 * TURN:
            pred = comem.comem_decode_saving_seconds(ctx_full[t], ctx_comem[t], s_bytes / 1e9, w_gbs) * 1e6
            rel.append(abs((t_full[t] - t_comem[t]) - pred) / pred)
    # overlap: memory-model decode attention on stream B under the agent's next steps on stream A
    overlap = []
    for t in range(T - 1):
        if not mem_in[t] or len(overlap) >= 4 and t < T - K - 1:
            continue
        reps = 6
        with torch.cuda.stream(sb):
            lens_m.fill_(mem_in[t])
        with torch.cuda.stream(sa):
            lens_a.fill_(ctx_comem[t + 1])
        torch.cuda.synchronize()
        for _ in range(4 * reps):
            launch(memory, lens_m, out_m, ws_m, sb)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(sa)
        for _ in range(reps):
            launch(agent, lens_a, out_a, ws_a, sa)
        e1.record(sa)
        torch.cuda.synchronize()
        e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e2.record(sa)
        for _ in range(reps):
            launch(agent, lens_a, out_a, ws_a, sa)
        e3.record(sa)
        torch.cuda.synchronize()
        rec = {"after_step": t + 1, "memory_ctx": mem_in[t], "agent_ctx": ctx_comem[t + 1],
               "agent_us_overlapped": e0.elapsed_time(e1) * 1e3 / reps,
               "agent_us_alone": e2.elapsed_time(e3) * 1e3 / reps, "sm_partition": []}
        # SM partitioning: both kernels are persistent one-CTA-per-SM grids, so two full grids time-share the GPU
        # and a short agent step queues behind a long memory step.  Giving each stream a share of the SMs
        # (per-call comem_launch_opts.grid_ctas, programmatic launch off so that a stream's next kernel does not park
        # on the other's SMs) lets both grids be resident at once.  The split is the library's policy
        # (comem_sm_partition: proportional to the bytes each batch streams); sms/4 and sms/2 are shown beside it.
        sms = comem.comem_grid_ctas(128)
        by_a = ctx_comem[t + 1] * CONC * agent.num_kv_heads * agent.head_dim * 4
        by_m = mem_in[t] * CONC * memory.num_kv_heads * memory.head_dim * 4
        pol_a, _ = comem.comem_sm_partition(by_a, by_m, sms)
        for agent_sms, how in ((pol_a, "comem_sm_partition"), (sms // 4, "fixed"), (sms // 2, "fixed")):
            for _ in range(4 * reps):
                comem.comem_decode_attn_async(memory.q, memory.k_pages, memory.v_pages, memory.block_table, lens_m,
                                              memory.softmax_scale, out_m, ws_m, stream=sb,
                                              grid_ctas=sms - agent_sms, programmatic_launch=False)
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(sa)
            for _ in range(reps):
                comem.comem_decode_attn_async(agent.q, agent.k_pages, agent.v_pages, agent.block_table, lens_a,
                                              agent.softmax_scale, out_a, ws_a, stream=sa,
                                              grid_ctas=agent_sms, programmatic_launch=False)
            p1.record(sa)
            torch.cuda.synchronize()
            rec["sm_partition"].append({"agent_sms": agent_sms, "memory_sms": sms - agent_sms, "split": how,
                                        "agent_us": p0.elapsed_time(p1) * 1e3 / reps})
        overlap.append(rec)
    del flush, out_a, out_m, ws_a, ws_m, agent, memory
    torch.cuda.empty_cache()
    # the whole trajectory through the library's scheduler, attention AND prefill per step; eq. 6 against it
    Y, YM = 32, 32
    traj = pipeline_trajectory(torch, comem, W, device, K, T, TURN, SUMM, CONC, Y, YM)
    p_tok_s = None
    unc_ms = traj["comem_memory_elsewhere"]["mean_ms_steps_with_uncached_prefill"]
    if unc_ms:
        # P of eq. 6: prompt tokens per second of the uncached prefill (summary + buffered turns, all sequences)
        l_sum_tokens = statistics.mean(c for c, e in zip(ctx_comem, events) if e.prefill_uncached)
        dec_ms = Y * statistics.mean(t_comem) / 1e3
        p_tok_s = CONC * l_sum_tokens / max((unc_ms - dec_ms) * 1e-3, 1e-9)
        l_full_mean, l_sum_mean = statistics.mean(ctx_full), statistics.mean(ctx_comem)
        traj["eq6"] = {"P_tokens_per_s": p_tok_s, "W_gbs": w_gbs, "Y_tokens_per_cycle": Y * K * CONC,
                       "L_full_mean": l_full_mean, "L_sum_mean": l_sum_mean,
                       "predicted_net_speedup": bool(comem.comem_net_speedup(Y * K, l_full_mean, l_sum_mean, s_bytes / 1e9, w_gbs,
                                                                             p_tok_s / CONC)),
                       "measured_net_speedup": traj["speedup_agent_stream"] > 1.0,
                       "max_compression_ratio_eq7": comem.comem_max_compression_ratio(w_gbs, Y * K, s_bytes / 1e9, p_tok_s / CONC)}
    print(json.dumps({
        "extra": "k-step-off pipeline (Algorithm 1) driven from comem_kstep_plan; eq. 5 vs measured",
        "trajectory": traj,
        "k": K, "steps": T, "turn_tokens": TURN, "summary_tokens": SUMM, "concurrency": CONC,
        "uncached_prefills": sum(int(e.prefill_uncached) for e in events),
        "memory_launches": sum(int(e.launch_memory) for e in events),
        "ctx_comem_min_max": [min(ctx_comem), max(ctx_comem)], "ctx_full_final": ctx_full[-1],
        "decode_attn_us_comem_sum": sum(t_comem), "decode_attn_us_full_sum": sum(t_full),
        "trajectory_speedup": sum(t_full) / sum(t_comem),
        "peak_step_speedup": max(f / c for f, c in zip(t_full, t_comem)),
        "fit": {"us_per_token": slope, "fixed_us": fixed, "W_gbs": w_gbs, "S_bytes_per_token": s_bytes},
        "eq5_rel_err": {"mean": sum(rel) / max(len(rel), 1), "max": max(rel) if rel else None, "steps": len(rel)},
        "per_step_us": {"comem": [round(x, 2) for x in t_comem], "full": [round(x, 2) for x in t_full]},
        "overlap": overlap, "l2": "flushed (512 MiB written) before every timed launch"}), flush=True)
    return 0


def load_peaks():
    peaks = {"hbm_gbs": FALLBACK_PEAK_GBS, "hbm_src": "fallback (B200_PROFILING.md)",
             "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "tf_src": "fallback (B200_PROFILING.md)"}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            m = json.load(f)
        peaks.update({"hbm_gbs": float(m["hbm_gbs"]), "hbm_src": "measured (MEASURED_PEAKS.json hbm_gbs, copy)",
                      "bf16_tflops": float(m["bf16_tflops"]), "bf16_tflops_sustained": float(m["bf16_tflops_sustained"]),
                      "tf_src": "measured (MEASURED_PEAKS.json)"})
    except Exception:  # noqa: BLE001
        pass
    return peaks


def measure_read_ceiling(torch, comem, device, stream, buf=None) -> dict:
    """what a read-only stream gets on this part -- the library's two hand-written sum-reductions
    (comem_read_ceiling_async) over >= 8 GiB, best of 5 each, CUDA events on the launch stream."""
    own = buf is None
    if own:
        buf = torch.empty(8 << 30, dtype=torch.uint8, device=device)
        buf.random_(0, 255)
    nbytes = (buf.numel() * buf.element_size()) // 8192 * 8192
    sink = torch.zeros(comem.COMEM_READ_CEILING_SINK_WORDS, dtype=torch.int64, device=device)
    out = {"bytes": nbytes}
    with torch.cuda.stream(stream):
        for variant, name in ((0, "vector_loads"), (1, "tma_ring")):
            ts = []
            for i in range(7):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                comem.comem_read_ceiling_async(buf, sink, variant, stream=stream, nbytes=nbytes)
                e1.record(stream)
                stream.synchronize()
                if i >= 2:
                    ts.append(e0.elapsed_time(e1))
            out[name + "_gbs"] = nbytes / min(ts) / 1e6
            out[name + "_gbs_median"] = nbytes / sorted(ts)[len(ts) // 2] / 1e6
    out["read_ceiling_gbs"] = max(out["vector_loads_gbs"], out["tma_ring_gbs"])
    return out


def measure_decode(ctx, name, steps, warmup, *, primary):
    """One decode workload: the timed K steps (graph replays), and -- for the primary workload -- the split-only
    timing, the isolated-step spread, a sustained run and the end-to-end leg."""
    torch, comem, replicas, args = ctx["torch"], ctx["comem"], ctx["replicas"], ctx["args"]
    device, rank, world, stream = ctx["device"], ctx["rank"], ctx["world"], ctx["stream"]
    R_spare = 8 if name == "c2" else 1
    spare = ((steps + max(warmup, 3)) // R_spare + 8) if primary else 0
    pools = make_pools(name, device, rank, spare)
    R = len(pools)
    outs = [torch.empty_like(b.q) for b in pools]
    ws = comem.alloc_workspace(pools[0].q, pools[0].k_pages, pools[0].block_table, stream=stream)
    step_bytes = [b.algorithmic_bytes() for b in pools]
    kv_pool_bytes = sum(int(b.seq_lens.sum().item()) * b.num_kv_heads * b.head_dim * 4 for b in pools)
    sampler = ClockSampler(str(getattr(torch.cuda.get_device_properties(device), 'uuid', '')), ctx["local_rank"])
    sampler.start()
    both = comem.COMEM_PHASE_SPLIT | comem.COMEM_PHASE_COMBINE
    use_graph = not args.no_graph
    flags = DEFAULT_LAUNCH_FLAGS if args.launch_flags is None else args.launch_flags
    res_flags = flags
    with torch.cuda.stream(stream):   # one checked step on pool 0 first (feeds the parity block): same launch flags
        comem.comem_decode_attn_async(pools[0].q, pools[0].k_pages, pools[0].v_pages, pools[0].block_table,
                                      pools[0].seq_lens, pools[0].softmax_scale, outs[0], ws, stream=stream, flags=flags)
    stream.synchronize()
    first_out = outs[0].clone()

    ms = timed_steps(torch, comem, replicas, pools, outs, ws, stream, steps, warmup, both, use_graph, sampler, device,
                     flags=flags)
    clocks = sampler.summary()
    bytes_k_steps = sum(step_bytes[i % R] for i in range(steps))
    ms_max = replicas.max_over_ranks(ms, device)
    total_bytes = replicas.sum_over_ranks(bytes_k_steps, device)
    res = {"pools": pools, "ws": ws, "R": R, "ms_max": ms_max, "total_bytes": total_bytes, "bytes_k_steps": bytes_k_steps,
           "kv_pool_bytes": kv_pool_bytes, "clocks": clocks, "first_out": first_out, "steps": steps,
           "launch_flags": res_flags}
    if primary:
        ms_split = timed_steps(torch, comem, replicas, pools, outs, ws, stream, steps, warmup,
                               comem.COMEM_PHASE_SPLIT, use_graph, sampler, device, flags=flags & 5)
        res["ms_split_max"] = replicas.max_over_ranks(ms_split, device)
        res["dist"] = step_distribution(torch, comem, pools, outs, ws, stream, 200 if name == "c2" else 20, both)
        # a sustained run of the same steps (seconds-scale thermals and the power cap show only here)
        long_steps = max(steps, 8192 if name == "c2" else 256)
        if long_steps != steps:
            sampler.reset()
            ms_long = timed_steps(torch, comem, replicas, pools, outs, ws, stream, long_steps, 3, both, use_graph,
                                  sampler, device, flags=flags)
            res["sustained"] = {"steps": long_steps, "us_per_step": replicas.max_over_ranks(ms_long, device) / long_steps * 1e3,
                                "clocks": sampler.summary()}
    sampler.stop()
    return res


def measure_fp8(ctx, peaks, steps, with_parity=True) -> dict:
    """The FP8 (E4M3 + page scales) cache on C4's batch, HND pools: the warp-level kernel (F2FP + HMMA, launch flags of the
    line) and the tcgen05 kernel (COMEM_LAUNCH_FP8_TENSOR), `steps` steps each from one replayed CUDA graph (a step reads
    4 GiB: cold in L2), parity of each against the FP8 oracle on one whole sequence."""
    torch, comem, args = ctx["torch"], ctx["comem"], ctx["args"]
    device, stream = ctx["device"], ctx["stream"]
    from paper_2605_30842_b200 import workloads as W

    bf = make_pools("c4", device, 0, 0)[0]
    f = W.to_hnd(W.quantize_batch_fp8(bf))
    del bf
    torch.cuda.empty_cache()
    nbytes = f.algorithmic_bytes()
    out = torch.empty_like(f.q)
    ws = comem.alloc_workspace(f.q, f.k_pages, f.block_table, stream=stream, kv_layout=f.kv_layout)
    res = {"workload": workload_desc("c4")["workload"] + ", cache quantised to E4M3 + per-page scales, HND pools",
           "algorithmic_bytes_per_step": nbytes, "steps": steps, "unit": UNIT, "launch": "CUDA graph, replayed"}
    # (the warp-level kernel in the classic order: a 0.65 ms step has nothing for the early mode to hide, and the FP8
    # consumers, bound by their issue slots, pay 5 % for its tests in the tile loop)
    for key, flags in (("warp_level", 0), ("tcgen05", comem.COMEM_LAUNCH_FP8_TENSOR)):
        sampler = ClockSampler(str(getattr(torch.cuda.get_device_properties(device), 'uuid', '')), ctx["local_rank"])
        sampler.start()
        with torch.cuda.stream(stream):
            def step():
                comem.comem_decode_attn_fp8_async(f.q, f.k_pages, f.v_pages, f.k_scale, f.v_scale, f.block_table,
                                                  f.seq_lens, f.softmax_scale, out, ws, stream=stream,
                                                  kv_layout=f.kv_layout, flags=flags)
            for _ in range(3):
                step()
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                for _ in range(steps):
                    step()
            g.replay()
            stream.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            sampler.active = True
            e0.record(stream)
            g.replay()
            e1.record(stream)
            stream.synchronize()
            sampler.active = False
            clocks = sampler.summary()
            us = e0.elapsed_time(e1) * 1e3 / steps
            # ... and sustained: the same graph replayed for ~1.5 s (this kernel plus HBM at full rate reaches the board's
            # power cap, the SM clock drops, and the two kernels part ways)
            reps = max(2, int(1.5e6 / (us * steps)))
            sampler.reset()
            sampler.active = True
            e0.record(stream)
            for _ in range(reps):
                g.replay()
            e1.record(stream)
            stream.synchronize()
            sampler.active = False
        sampler.stop()
        us_long = e0.elapsed_time(e1) * 1e3 / (steps * reps)
        gbs = nbytes / us / 1e3
        rec = {"kernel": "decode_fp8_tc_kernel" if flags & 8 else "decode_split_kernel<128, 1, %d>" % (flags & 1), "launch_flags": flags,
               "us_per_step": us, "achieved": gbs, "frac": gbs / peaks["hbm_gbs"], "frac_of_8TBps": gbs / 8000.0,
               "gpu_launches": steps * (2 if flags & 8 else 1), "clocks": clocks,
               "traffic": ncu_traffic("fp8tc_c4_hnd" if flags & 8 else "fp8_c4_hnd"),
               "sustained": {"steps": steps * reps, "us_per_step": us_long, "achieved": nbytes / us_long / 1e3,
                             "frac": nbytes / us_long / 1e3 / peaks["hbm_gbs"], "clocks": sampler.summary()}}
        if with_parity:
            rec["parity"], _ = fp8_parity(f, out, seq=3)
        res[key] = rec
        del g
    return res


def measure_prefill(ctx, peaks, with_parity=True) -> dict:
    """the paged causal prefill kernel (tcgen05) on the agent geometry -- an uncached full prefill
    of one 32 768-token context (Alg. 1 line 12) and a cached 512-token chunk over the same prefix (line 10).
    TFLOP/s = causal flops (4 D per (query, key <= pos) pair and query head) / CUDA-event time, against the measured
    sustained bf16 peak."""
    torch, comem, stream = ctx["torch"], ctx["comem"], ctx["stream"]
    from paper_2605_30842_b200 import workloads as W

    out = {}
    for key, lens, qn in (("uncached_32k", [32768], [32768]), ("cached_chunk_512_over_32k", [32768], [512]),
                          ("batch8_uncached_8k", [8192] * 8, [8192] * 8)):
        pb = W.make_prefill_batch(lens, qn, 64, 8, 128, 16, seed=2001, device=ctx["device"], k_scale=0.5)
        o = torch.empty_like(pb.q)
        reps = 3 if key == "uncached_32k" else 10
        with torch.cuda.stream(stream):
            f = lambda: comem.comem_prefill_attn_async(pb.q, pb.k_pages, pb.v_pages, pb.block_table, pb.seq_lens,  # noqa: E731
                                                       pb.q_start, pb.softmax_scale, o, stream=stream)
            for _ in range(3):
                f()
            stream.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                f()
            e1.record(stream)
            stream.synchronize()
        ms = e0.elapsed_time(e1) / reps
        fl = pb.algorithmic_flops()
        rec = {"ms": ms, "algorithmic_flops": fl, "tflops": fl / ms / 1e9,
               "frac_of_sustained_peak": fl / ms / 1e9 / peaks["bf16_tflops_sustained"],
               "frac_of_burst_peak": fl / ms / 1e9 / peaks["bf16_tflops"]}
        if key == "uncached_32k":
            rec["tokens_per_s"] = 32768 / (ms * 1e-3)
        if with_parity and key != "batch8_uncached_8k":
            rec["parity"] = prefill_parity_sampled(pb, o)
        out[key] = rec
        del pb, o
    return out


def prefill_parity_sampled(pb, gpu_out, n_rows=6):
    """Oracle on sampled query rows of a prefill batch, all query heads: row i of sequence 0 is, by the prefill
    oracle's own definition (pin PF2), the decode oracle on the cache truncated at its position."""
    import numpy as np
    import torch
    import oracle

    oracle.build()
    L, n = int(pb.seq_lens[0]), int(pb.q_start[1])
    rows = sorted({0, 1, n // 3, n // 2 + 5, n - 2, n - 1} & set(range(n)))[:n_rows]
    ps = pb.page_size
    npg = (L + ps - 1) // ps
    ids = pb.block_table[0, :npg].long()
    kp, vp = pb.k_pages[ids].cpu(), pb.v_pages[ids].cpu()
    bt = torch.arange(npg, dtype=torch.int32).view(1, npg).repeat(len(rows), 1)
    sl = torch.tensor([L - n + i + 1 for i in rows], dtype=torch.int32)
    q = pb.q[rows].cpu().contiguous()
    ref, _ = oracle.decode_attn(q, kp, vp, bt, sl, pb.softmax_scale)
    got = gpu_out[rows].double().cpu().numpy()
    d = np.abs(got - ref)
    par = {"rows": len(rows) * pb.num_q_heads, "max_abs": float(d.max()), "mean_abs": float(d.mean()),
           "rel_l2": float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300))}
    par["ok"] = bool(par["max_abs"] <= 2e-2 and par["mean_abs"] <= 2e-3 and par["rel_l2"] <= 5e-3)
    return par


def run_prefill(args) -> int:
    """--prefill: the prefill kernel's own JSON line (extra; metric TFLOP/s against the measured bf16 peak)."""
    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build

    device = torch.device("cuda", 0)
    torch.cuda.set_device(device)
    cuda_build.build()
    comem.load_library()
    peaks = load_peaks()
    ctx = {"torch": torch, "comem": comem, "device": device, "stream": torch.cuda.Stream(device)}
    sampler = ClockSampler(str(getattr(torch.cuda.get_device_properties(device), 'uuid', '')), 0)
    sampler.start()
    sampler.active = True
    pf = measure_prefill(ctx, peaks, with_parity=not args.no_cpu_baseline)
    sampler.active = False
    sampler.stop()
    top = pf["uncached_32k"]
    print(json.dumps({"extra": "paged causal prefill attention (tcgen05)", "metric": "prefill_attn_tflops",
                      "value": top["tflops"], "unit": "TFLOP/s", "dtype": "bf16", "data": "synthetic",
                      "config": {"workload": "uncached full prefill: batch 1, 64q/8kv, D128, 32768 tokens, page 16"},
                      "roofline": {"bound": "tensor", "kernel": "prefill_attn_kernel<128>", "achieved": top["tflops"],
                                   "peak": peaks["bf16_tflops_sustained"], "peak_source": peaks["tf_src"] + " bf16_tflops_sustained",
                                   "unit": "TFLOP/s", "frac": top["frac_of_sustained_peak"],
                                   "traffic": ncu_traffic("prefill_uncached_32k")},
                      "prefill": pf, "clocks": sampler.summary()}), flush=True)
    return 0


def main() -> int:
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank)
    if args.window > 0:
        return run_window(args) if rank == 0 else 0
    if args.offload:
        return run_offload(args) if rank == 0 else 0
    if args.pipeline > 0:
        return run_pipeline(args) if rank == 0 else 0
    if args.kv_fp8:
        return run_fp8(args) if rank == 0 else 0
    if args.affine:
        return run_affine(args) if rank == 0 else 0
    if args.prefill:
        return run_prefill(args) if rank == 0 else 0
    if args.workload == "c5":
        return run_c5(args) if rank == 0 else 0

    import torch
    import paper_2605_30842_b200 as comem
    from paper_2605_30842_b200 import build as cuda_build
    from paper_2605_30842_b200 import replicas

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback exists)"
    rank, local_rank, world = replicas.init("nccl")
    assert world == args.gpus or world == 1, f"--gpus {args.gpus} but WORLD_SIZE={world}"
    device = torch.device("cuda", local_rank)
    torch.cuda.set_device(device)
    if rank == 0:
        cuda_build.build()
    replicas.barrier()
    comem.load_library()
    peaks = load_peaks()
    stream = torch.cuda.Stream(device)
    ctx = {"torch": torch, "comem": comem, "replicas": replicas, "args": args, "device": device, "rank": rank,
           "local_rank": local_rank, "world": world, "stream": stream}

    prim = measure_decode(ctx, args.workload, args.steps, args.warmup, primary=True)
    pools, ws, R = prim["pools"], prim["ws"], prim["R"]
    cpu_base, parity = None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_base, parity = cpu_baseline_and_parity(pools[0], prim["first_out"])
    e2e_sampler = ClockSampler(str(getattr(torch.cuda.get_device_properties(device), 'uuid', '')), local_rank)
    e2e_sampler.start()
    e2e_ms, e2e_bytes, h2d, d2h = timed_e2e(torch, comem, replicas, pools, ws, stream, args.steps, args.warmup,
                                            e2e_sampler, device, 5000 + 1000 * rank)
    e2e_sampler.stop()
    e2e_ms_max = replicas.max_over_ranks(e2e_ms, device)
    e2e_total = replicas.sum_over_ranks(e2e_bytes, device)
    checks = pools[0].checksums()
    del pools, ws
    prim["pools"] = prim["ws"] = None
    torch.cuda.empty_cache()

    # The other workloads the metric is quoted on ("at 32K-128K ctx"): C3, C4, C5's aggregate, the prefill kernel and
    # the read-only ceiling, inside the same JSON line (1 GPU, default workload only; --primary-only skips them).
    extra = {}
    ceiling = None
    if rank == 0 and world == 1 and args.workload == "c2" and not args.primary_only:
        for name in ("c3", "c4"):
            k = max(3, min(args.steps, 100))
            r = measure_decode(ctx, name, k, 3, primary=False)
            us = r["ms_max"] / k * 1e3
            gbs = (r["bytes_k_steps"] / k) / us / 1e3
            rec = {"workload": workload_desc(name)["workload"], "steps": k, "us_per_step": us, "achieved": gbs,
                   "unit": UNIT, "frac": gbs / peaks["hbm_gbs"], "frac_of_8TBps": gbs / 8000.0,
                   "algorithmic_bytes_per_step": r["bytes_k_steps"] // k, "traffic": ncu_traffic(name),
                   "launch": "CUDA graph, replayed", "clocks": r["clocks"]}
            if not args.no_cpu_baseline:
                cb, par = cpu_baseline_and_parity(r["pools"][0], r["first_out"], budget_s=6.0)
                rec["parity"] = par
                rec["oracle_gbs"] = cb["value"]
            extra[name] = rec
            r["pools"] = r["ws"] = None
            del r
            torch.cuda.empty_cache()
        ceiling = measure_read_ceiling(torch, comem, device, stream)   # its own 8 GiB buffer
        torch.cuda.empty_cache()
        for rec in extra.values():
            rec["frac_of_read_ceiling"] = rec["achieved"] / ceiling["read_ceiling_gbs"]
        c5 = measure_c5(args, torch, comem, device, reps=2)
        c5["frac_of_8TBps"] = c5["aggregate_gbs"] / 8000.0
        c5["frac_of_read_ceiling"] = c5["aggregate_gbs"] / ceiling["read_ceiling_gbs"]
        extra["c5"] = c5
        torch.cuda.empty_cache()
        extra["prefill"] = measure_prefill(ctx, peaks, with_parity=not args.no_cpu_baseline)
        torch.cuda.empty_cache()
        extra["c4_fp8"] = measure_fp8(ctx, peaks, max(3, min(args.steps, 100)), with_parity=not args.no_cpu_baseline)
        for k_ in ("warp_level", "tcgen05"):
            extra["c4_fp8"][k_]["frac_of_read_ceiling"] = extra["c4_fp8"][k_]["achieved"] / ceiling["read_ceiling_gbs"]
        torch.cuda.empty_cache()

    if rank == 0:
        peak, peak_src = peaks["hbm_gbs"], peaks["hbm_src"]
        ms_max, steps = prim["ms_max"], args.steps
        value = prim["total_bytes"] / (ms_max * 1e-3) / 1e9
        achieved = (prim["bytes_k_steps"] / steps) / (ms_max / steps * 1e-3) / 1e9
        cfg = workload_desc(args.workload)
        kvp = prim["kv_pool_bytes"]
        a, r_ = divmod(steps, R)
        cfg.update({"l2": (f"cold: steps rotate over {R} disjoint KV pools ({kvp / 2**30:.2f} GiB) > L2"
                           if R > 1 else f"cold: one step reads {kvp / 2**30:.2f} GiB of KV >> L2"),
                    "launch": ("CUDA graphs only: %d replays of a %d-step graph + one %d-step graph" % (a, R, r_))
                    if not args.no_graph else "host launches",
                    "algorithmic_bytes_per_step": prim["bytes_k_steps"] // steps,
                    "grid_ctas": comem.comem_grid_ctas(cfg["head_dim"]),
                    "replicas": world})
        roof = {"bound": "hbm", "kernel": "decode_split_kernel<128, 0, %d>" % (1 if prim["launch_flags"] & 1 else 0), "achieved": achieved,
                "peak": peak, "peak_source": peak_src, "unit": UNIT, "frac": achieved / peak,
                "us_per_launch": ms_max / steps * 1e3,
                "split_only_us": prim["ms_split_max"] / steps * 1e3,
                "traffic": ncu_traffic(args.workload), "traffic_source": "profiles/ncu_traffic.json (null when the capture predates the kernel sources)"}
        if ceiling is not None:
            roof["read_ceiling_gbs"] = ceiling["read_ceiling_gbs"]
            roof["frac_of_read_ceiling"] = achieved / ceiling["read_ceiling_gbs"]
            roof["read_ceiling"] = ceiling
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
                "warmup": args.warmup, "ms_per_step": ms_max / steps, "us_per_step": ms_max / steps * 1e3,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
                "data": "synthetic", "config": cfg,
                "frac_of_8TBps": value / world / 8000.0,
                "roofline": roof,
                "e2e": {"value": e2e_total / (e2e_ms_max * 1e-3) / 1e9, "unit": UNIT,
                        "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "us_per_step": e2e_ms_max / steps * 1e3,
                        "api": "comem_decode_step_host through the binding's pre-marshalled call object (DecodeStepHost), pinned host buffers: K3 reads the q,k,v rows over the host link and appends -> fused split+combine stores out into host memory -> stream synchronize (2 launches, no copy engine)"},
                "isolated_step_us": prim["dist"], "input_checksums": checks,
                "gpu_launches": steps * (2 if (prim["launch_flags"] & 2) and args.workload == "c2" else 1),
                "launch_flags": prim["launch_flags"],
                "clocks": prim["clocks"]}
        if "sustained" in prim:
            s_ = prim["sustained"]
            s_["achieved"] = (prim["bytes_k_steps"] / steps) / s_["us_per_step"] / 1e3
            s_["frac"] = s_["achieved"] / peak
            line["sustained"] = s_
        if cpu_base is not None:
            line["cpu_baseline"] = cpu_base
            line["parity"] = parity
        if extra:
            line["workloads"] = extra
        print(json.dumps(line), flush=True)
    replicas.finalize()
    return 0


if __name__ == "__main__":
    sys.exit(main())
