"""Per-CTA stage timeline of the split-KV kernel (development diagnostic, not a benchmark).

    python -m paper_2605_30842_b200.build --trace      # builds libcomem_decode_trace.so (-DCOMEM_TRACE)
    python -m paper_2605_30842_b200.stage_trace [c2|c2x4]

Runs 12 back-to-back launches (8 rotating pools, host launches) and has the LAST one stamp
%globaltimer at its stage boundaries; prints, per stage, min / median / max over the CTAs in ns
after the first CTA's entry, and the per-CTA stage durations.  The numbers carry the cost of the
stamps themselves (a few tens of ns each) and %globaltimer's 32 ns granularity.
"""
from __future__ import annotations

import ctypes
import sys

import numpy as np
import torch

from . import binding
from . import build as cuda_build
from . import workloads as W

STAGES = ["entry", "pdl_wait", "prefix", "first_data", "stream_done", "published", "ticket", "seg_done"]


def main(which: str = "c2") -> None:
    binding._LIB_PATH = cuda_build.TRACE_LIB
    binding._lib = None
    lib = binding.load_library()
    lib.comem_set_trace.argtypes = [ctypes.c_void_p]
    dev = "cuda"
    nseq = 4 if which == "c2x4" else 1
    pools = [W.make_batch([32768] * nseq, 64, 8, 128, 16, 1002 + i, dev, k_scale=0.5,
                          num_pages=4096 * nseq) for i in range(8)]
    outs = [torch.empty_like(b.q) for b in pools]
    ws = binding.alloc_workspace(pools[0].q, pools[0].k_pages, pools[0].block_table)
    grid = binding.comem_grid_ctas(128)
    trace = torch.zeros(grid * 16, dtype=torch.int64, device=dev)

    def run(n, phases):
        for i in range(n):
            b = pools[i % 8]
            binding.comem_decode_attn_phases_async(b.q, b.k_pages, b.v_pages, b.block_table, b.seq_lens,
                                                   b.softmax_scale, outs[i % 8], ws, phases=phases)

    both = binding.COMEM_PHASE_SPLIT | binding.COMEM_PHASE_COMBINE
    for label, ph in (("fused", both), ("split-only", binding.COMEM_PHASE_SPLIT)):
        lib.comem_set_trace(None)
        run(16, ph)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        run(64, ph)
        e1.record()
        torch.cuda.synchronize()
        print(f"{which} {label}: {e0.elapsed_time(e1) / 64 * 1e3:.2f} us/launch (host launches, back to back)")
        trace.zero_()
        torch.cuda.synchronize()
        run(11, ph)
        lib.comem_set_trace(ctypes.c_void_p(trace.data_ptr()))
        run(1, ph)
        torch.cuda.synchronize()
        t = trace.cpu().numpy().reshape(grid, 16).astype(np.int64)
        t0 = t[:, 0][t[:, 0] > 0].min()
        print("  stage            min     p50     max   ns after the first CTA's entry")
        for i, nm in enumerate(STAGES):
            col = t[:, i][t[:, i] > 0] - t0
            if len(col):
                print(f"  {nm:12s} {col.min():7d} {int(np.median(col)):7d} {col.max():7d}   n={len(col)}")
        for i in range(7):
            ok = (t[:, i] > 0) & (t[:, i + 1] > 0)
            if ok.any():
                d = (t[:, i + 1] - t[:, i])[ok]
                print(f"  d {STAGES[i]:>12s} -> {STAGES[i + 1]:12s} p50 {int(np.median(d)):6d}  max {d.max():6d}")
        ok = (t[:, 10] > 0) & (t[:, 6] > 0)
        if ok.any():
            for nm, c in (("ticket -> loads issued, scalars back", t[:, 8] - t[:, 6]),
                          ("-> cp.async rows landed", t[:, 9] - t[:, 8]),
                          ("-> accumulated", t[:, 10] - t[:, 9]), ("-> stored + barrier", t[:, 7] - t[:, 10])):
                print(f"  merge {nm:38s} p50 {int(np.median(c[ok])):6d}  max {c[ok].max():6d}  n={ok.sum()}")


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "c2")
