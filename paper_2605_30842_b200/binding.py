"""Thin ctypes binding over libcomem_decode.so — same names as include/comem_decode_attn.h.

Argument marshalling only: shapes are read off the tensors, pointers are
``tensor.data_ptr()``, the stream is torch's current CUDA stream unless given.
Every step of the path runs in the library's kernels; there is no fallback —
if the library is missing or the device is not sm_100 the call raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcomem_decode.so")
_lib = None

COMEM_OK = 0
COMEM_ERR_INVALID_ARG = 1
COMEM_ERR_UNSUPPORTED = 2
COMEM_ERR_WORKSPACE = 3
COMEM_ERR_CUDA = 4


class ComemError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {comem_status_string(status)} (status {status})")


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen the C-ABI library (built in-tree by ``python -m paper_2605_30842_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2605_30842_b200.build` "
            "(or __graft_entry__.build()). There is no CPU or PyTorch fallback for this path.")
    lib = ctypes.CDLL(_LIB_PATH)
    c = ctypes
    vp, i32, i64, f32, sz = c.c_void_p, c.c_int, c.c_int64, c.c_float, c.c_size_t
    lib.comem_decode_attn_async.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32, i32,
                                            i64, vp, vp, sz, vp, vp]
    lib.comem_decode_attn_async.restype = i32
    lib.comem_decode_attn_static_async.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32, i32,
                                                   i64, vp, vp, vp]
    lib.comem_decode_attn_static_async.restype = i32
    lib.comem_static_scratch_bytes.argtypes = []
    lib.comem_static_scratch_bytes.restype = sz
    lib.comem_decode_attn_phases_async.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32,
                                                   i32, i64, vp, vp, sz, vp, i32, vp]
    lib.comem_decode_attn_phases_async.restype = i32
    lib.comem_decode_attn_window_async.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32,
                                                   i32, i64, vp, vp, sz, vp, i32, i32, vp]
    lib.comem_decode_attn_window_async.restype = i32
    lib.comem_decode_attn_fp8_async.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32,
                                                i32, i64, vp, vp, sz, vp, i32, i32, i32, vp]
    lib.comem_decode_attn_fp8_async.restype = i32
    lib.comem_decode_attn_offload_async.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32, i32,
                                                    i64, i64, vp, vp, sz, vp, vp]
    lib.comem_decode_attn_offload_async.restype = i32
    lib.comem_pages_copy_async.argtypes = [vp, vp, vp, vp, vp, vp, i32, sz, vp]
    lib.comem_pages_copy_async.restype = i32
    lib.comem_kstep_step_async.argtypes = [vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.comem_kstep_step_async.restype = i32
    lib.comem_decode_step_host_fp8.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32, i32,
                                               i64, vp, vp, sz, vp, i32]
    lib.comem_decode_step_host_fp8.restype = i32
    lib.comem_prefill_attn_async.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32, i32, i32,
                                             i64, vp, vp, vp]
    lib.comem_prefill_attn_async.restype = i32
    lib.comem_decode_attn.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32, i32, i64,
                                      vp, vp, sz]
    lib.comem_decode_attn.restype = i32
    lib.comem_decode_attn_workspace_bytes.argtypes = [i32] * 6
    lib.comem_decode_attn_workspace_bytes.restype = sz
    lib.comem_workspace_init_async.argtypes = [vp, sz, i32, i32, i32, i32, vp]
    lib.comem_workspace_init_async.restype = i32
    lib.comem_validate_inputs.argtypes = [vp, vp, i32, i32, i32, i64, vp, sz, vp]
    lib.comem_validate_inputs.restype = i32
    lib.comem_kv_append_async.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp]
    lib.comem_kv_append_async.restype = i32
    lib.comem_kv_append_fp8_async.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp]
    lib.comem_kv_append_fp8_async.restype = i32
    lib.comem_decode_step_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, i32,
                                           i32, i64, vp, vp, sz, vp]
    lib.comem_decode_step_host.restype = i32
    f64 = c.c_double
    lib.comem_kstep_plan.argtypes = [i32, i32, i32, vp]
    lib.comem_kstep_plan.restype = i32
    lib.comem_kstep_context_lengths.argtypes = [vp, i32, i32, i32, vp, vp, vp]
    lib.comem_kstep_context_lengths.restype = i32
    lib.comem_decode_saving_seconds.argtypes = [f64] * 4
    lib.comem_decode_saving_seconds.restype = f64
    lib.comem_net_speedup.argtypes = [f64] * 6
    lib.comem_net_speedup.restype = i32
    lib.comem_max_compression_ratio.argtypes = [f64] * 4
    lib.comem_max_compression_ratio.restype = f64
    lib.comem_schedule_host.argtypes = [vp, i32, i32, i32, vp, vp]
    lib.comem_schedule_host.restype = i32
    lib.comem_grid_ctas.argtypes = [i32]
    lib.comem_grid_ctas.restype = i32
    lib.comem_read_ceiling_async.argtypes = [vp, sz, vp, i32, vp]
    lib.comem_read_ceiling_async.restype = i32
    lib.comem_sm_partition.argtypes = [f64, f64, i32, i32, vp, vp]
    lib.comem_sm_partition.restype = i32
    lib.comem_set_grid_ctas.argtypes = [i32]
    lib.comem_set_grid_ctas.restype = i32
    lib.comem_set_programmatic_launch.argtypes = [i32]
    lib.comem_set_programmatic_launch.restype = i32
    lib.comem_status_string.argtypes = [i32]
    lib.comem_status_string.restype = c.c_char_p
    lib.comem_version.restype = i32
    _lib = lib
    return lib


def comem_status_string(status: int) -> str:
    return load_library().comem_status_string(int(status)).decode()


def comem_version() -> int:
    return int(load_library().comem_version())


def comem_grid_ctas(head_dim: int) -> int:
    g = int(load_library().comem_grid_ctas(int(head_dim)))
    if g < 0:
        raise ComemError(-g, "comem_grid_ctas")
    return g


COMEM_LAUNCH_KV_PREFIX_IMMUTABLE = 1
COMEM_LAUNCH_SPLIT_COMBINE = 2
COMEM_LAUNCH_Q_STABLE = 4
COMEM_LAUNCH_FP8_TENSOR = 8


class LaunchOpts(ctypes.Structure):
    """comem_launch_opts: per-call grid size (0 = default), programmatic launch (-1 = default), COMEM_LAUNCH_* flags."""
    _fields_ = [("grid_ctas", ctypes.c_int), ("programmatic_launch", ctypes.c_int), ("flags", ctypes.c_int)]


def _opts(grid_ctas, programmatic_launch, flags=0):
    """None when all are defaults, else a pointer to a comem_launch_opts (the library reads it during the call)."""
    if grid_ctas is None and programmatic_launch is None and not flags:
        return None
    o = LaunchOpts(int(grid_ctas or 0), -1 if programmatic_launch is None else (1 if programmatic_launch else 0),
                   int(flags))
    return ctypes.cast(ctypes.pointer(o), ctypes.c_void_p)


def comem_sm_partition(bytes_a: float, bytes_b: float, num_sms: int, min_ctas: int = 8):
    """(ctas_a, ctas_b): the library's SM split for two batches sharing the GPU, proportional to their bytes."""
    a, b = ctypes.c_int(0), ctypes.c_int(0)
    st = load_library().comem_sm_partition(float(bytes_a), float(bytes_b), int(num_sms), int(min_ctas),
                                           ctypes.cast(ctypes.byref(a), ctypes.c_void_p),
                                           ctypes.cast(ctypes.byref(b), ctypes.c_void_p))
    if st != COMEM_OK:
        raise ComemError(st, "comem_sm_partition")
    return a.value, b.value


COMEM_READ_CEILING_SINK_WORDS = 1024


def comem_read_ceiling_async(buf: torch.Tensor, sink: torch.Tensor, variant: int = 0, stream=None, nbytes=None) -> None:
    """Measurement aid: enqueue the read-only sum-reduction over `buf` (variant 0: vector loads, 1: TMA ring)."""
    assert buf.is_cuda and buf.is_contiguous() and sink.is_cuda and sink.dtype == torch.int64
    assert sink.numel() >= COMEM_READ_CEILING_SINK_WORDS
    n = buf.numel() * buf.element_size() if nbytes is None else int(nbytes)
    st = load_library().comem_read_ceiling_async(_ptr(buf), n, _ptr(sink), int(variant), _stream(stream))
    if st != COMEM_OK:
        raise ComemError(st, "comem_read_ceiling_async")


def comem_set_grid_ctas(n: int) -> None:
    load_library().comem_set_grid_ctas(int(n))


def comem_set_programmatic_launch(enabled: bool) -> None:
    load_library().comem_set_programmatic_launch(1 if enabled else 0)


def comem_schedule_host(seq_lens, num_kv_heads: int, grid_ctas: int):
    """Host mirror of the device split-KV schedule: list of CTA tile-range boundaries."""
    import numpy as np

    sl = np.ascontiguousarray(np.asarray(seq_lens, dtype=np.int32))
    begins = np.zeros(grid_ctas + 1, dtype=np.int64)
    nc = ctypes.c_int(0)
    st = load_library().comem_schedule_host(sl.ctypes.data, len(sl), int(num_kv_heads), int(grid_ctas),
                                            begins.ctypes.data, ctypes.byref(nc))
    if st != COMEM_OK:
        raise ComemError(st, "comem_schedule_host")
    return begins[:nc.value + 1].tolist()


class KstepEvent(ctypes.Structure):
    _fields_ = [("step", ctypes.c_int32), ("summary_upto", ctypes.c_int32), ("adopt_summary", ctypes.c_uint8),
                ("prefill_uncached", ctypes.c_uint8), ("launch_memory", ctypes.c_uint8), ("reserved", ctypes.c_uint8)]


def comem_kstep_plan(num_steps: int, k: int, mem_delay: int = 0):
    """Algorithm 1 as a list of KstepEvent (host function of the library)."""
    ev = (KstepEvent * max(num_steps, 1))()
    st = load_library().comem_kstep_plan(int(num_steps), int(k), int(mem_delay), ctypes.cast(ev, ctypes.c_void_p))
    if st != COMEM_OK:
        raise ComemError(st, "comem_kstep_plan")
    return ev, [ev[i] for i in range(num_steps)]


class KstepModel(ctypes.Structure):
    """comem_kstep_model (include/comem_decode_attn.h)."""
    _fields_ = [(n, ctypes.c_void_p) for n in ("q_decode", "out_decode", "q_prefill", "out_prefill", "new_k", "new_v",
                                               "k_pages", "v_pages", "block_table", "seq_lens", "q_start", "workspace")] + \
               [("workspace_bytes", ctypes.c_size_t), ("num_pages", ctypes.c_int64), ("prefill_cap", ctypes.c_int64)] + \
               [(n, ctypes.c_int) for n in ("batch", "num_q_heads", "num_kv_heads", "head_dim", "page_size",
                                            "max_pages_per_seq")] + [("softmax_scale", ctypes.c_float)]


class KstepStepStats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("agent_ctx", "agent_prefill_tokens", "memory_ctx", "agent_grid",
                                              "memory_grid", "memory_in_flight", "launches")]


def kstep_model(q_decode, out_decode, q_prefill, out_prefill, new_k, new_v, k_pages, v_pages, block_table, seq_lens,
                q_start, workspace, softmax_scale: float) -> KstepModel:
    """Fill a comem_kstep_model from torch tensors (pointers only: keep the tensors alive)."""
    m = KstepModel()
    for name, t in (("q_decode", q_decode), ("out_decode", out_decode), ("q_prefill", q_prefill),
                    ("out_prefill", out_prefill), ("new_k", new_k), ("new_v", new_v), ("k_pages", k_pages),
                    ("v_pages", v_pages), ("block_table", block_table), ("seq_lens", seq_lens), ("q_start", q_start),
                    ("workspace", workspace)):
        assert t.is_cuda and t.is_contiguous()
        setattr(m, name, t.data_ptr())
    m.workspace_bytes = workspace.numel() * workspace.element_size()
    m.num_pages, m.prefill_cap = k_pages.shape[0], q_prefill.shape[0]
    m.batch, m.num_q_heads, m.head_dim = q_decode.shape
    m.num_kv_heads, m.page_size, m.max_pages_per_seq = k_pages.shape[2], k_pages.shape[1], block_table.shape[1]
    m.softmax_scale = float(softmax_scale)
    return m


def comem_kstep_step_async(event, turn_tokens: int, summary_tokens: int, decode_tokens: int, memory_decode_tokens: int,
                           agent: KstepModel, memory, agent_stream, memory_stream=None, memory_done_event=None,
                           agent_step_event=None) -> KstepStepStats:
    """One agent step of Algorithm 1 enqueued by the library's scheduler (see the header).  `event`: one
    comem_kstep_event of comem_kstep_plan's array; events: torch.cuda.Event objects that have been recorded once
    (so that their CUDA handle exists), or None."""
    stats = KstepStepStats()
    ev = lambda e: None if e is None else ctypes.c_void_p(e.cuda_event)  # noqa: E731
    st = load_library().comem_kstep_step_async(
        ctypes.byref(event), int(turn_tokens), int(summary_tokens), int(decode_tokens), int(memory_decode_tokens),
        ctypes.byref(agent), None if memory is None else ctypes.byref(memory), _stream(agent_stream),
        None if memory_stream is None else _stream(memory_stream), ev(memory_done_event), ev(agent_step_event),
        ctypes.byref(stats))
    if st != COMEM_OK:
        raise ComemError(st, "comem_kstep_step_async")
    return stats


def comem_kstep_context_lengths(events_array, num_steps: int, turn_tokens: int, summary_tokens: int):
    """(comem_ctx, full_ctx, memory_input) token counts per step, as python lists."""
    a, b, c_ = ((ctypes.c_int32 * max(num_steps, 1))() for _ in range(3))
    st = load_library().comem_kstep_context_lengths(ctypes.cast(events_array, ctypes.c_void_p), int(num_steps),
                                                    int(turn_tokens), int(summary_tokens),
                                                    ctypes.cast(a, ctypes.c_void_p), ctypes.cast(b, ctypes.c_void_p),
                                                    ctypes.cast(c_, ctypes.c_void_p))
    if st != COMEM_OK:
        raise ComemError(st, "comem_kstep_context_lengths")
    return list(a)[:num_steps], list(b)[:num_steps], list(c_)[:num_steps]


def comem_decode_saving_seconds(l_full, l_sum, s_gb_per_token, w_gb_per_s) -> float:
    return float(load_library().comem_decode_saving_seconds(l_full, l_sum, s_gb_per_token, w_gb_per_s))


def comem_net_speedup(y_tokens, l_full, l_sum, s_gb_per_token, w_gb_per_s, p_tokens_per_s) -> bool:
    return bool(load_library().comem_net_speedup(y_tokens, l_full, l_sum, s_gb_per_token, w_gb_per_s, p_tokens_per_s))


def comem_max_compression_ratio(w_gb_per_s, y_tokens, s_gb_per_token, p_tokens_per_s) -> float:
    return float(load_library().comem_max_compression_ratio(w_gb_per_s, y_tokens, s_gb_per_token, p_tokens_per_s))


def comem_decode_attn_workspace_bytes(batch: int, num_q_heads: int, num_kv_heads: int, head_dim: int,
                                      page_size: int, max_pages_per_seq: int) -> int:
    return int(load_library().comem_decode_attn_workspace_bytes(
        int(batch), int(num_q_heads), int(num_kv_heads), int(head_dim), int(page_size),
        int(max_pages_per_seq)))


def comem_workspace_init_async(workspace: torch.Tensor, batch: int, num_q_heads: int, num_kv_heads: int,
                               head_dim: int, stream=None) -> None:
    st = load_library().comem_workspace_init_async(_ptr(workspace), workspace.numel(), int(batch),
                                                   int(num_q_heads), int(num_kv_heads), int(head_dim),
                                                   _stream(stream))
    if st != COMEM_OK:
        raise ComemError(st, "comem_workspace_init_async")


def alloc_workspace(q: torch.Tensor, k_pages: torch.Tensor, block_table: torch.Tensor, stream=None,
                    kv_layout: str = "NHD") -> torch.Tensor:
    """torch.empty of the size the library asks for (device memory is torch's job), then the
    library's one-time comem_workspace_init_async on it (on `stream` or the current stream)."""
    ps, hkv = (k_pages.shape[2], k_pages.shape[1]) if kv_layout == "HND" else (k_pages.shape[1], k_pages.shape[2])
    n = comem_decode_attn_workspace_bytes(q.shape[0], q.shape[1], hkv, q.shape[2], ps, block_table.shape[1])
    ws = torch.empty(n, dtype=torch.uint8, device=q.device)
    with torch.cuda.device(q.device):
        if isinstance(stream, torch.cuda.Stream):
            # torch's caching allocator hands out blocks that are free in CURRENT-stream order: work queued there
            # may still be writing this block's previous contents.  The init below runs on `stream`, so order it
            # after the current stream and tell the allocator where the block is used.
            stream.wait_stream(torch.cuda.current_stream())
            ws.record_stream(stream)
        comem_workspace_init_async(ws, q.shape[0], q.shape[1], hkv, q.shape[2], stream)
    return ws


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    if isinstance(stream, torch.cuda.Stream):
        return ctypes.c_void_p(stream.cuda_stream)
    return ctypes.c_void_p(int(stream))


def _check_inputs(q, k_pages, v_pages, block_table, seq_lens):
    assert q.dtype == torch.bfloat16 and k_pages.dtype == torch.bfloat16 and v_pages.dtype == torch.bfloat16
    assert block_table.dtype == torch.int32 and seq_lens.dtype == torch.int32
    assert q.is_contiguous() and k_pages.is_contiguous() and v_pages.is_contiguous()
    assert block_table.is_contiguous() and seq_lens.is_contiguous()
    assert q.dim() == 3 and k_pages.dim() == 4 and k_pages.shape == v_pages.shape
    assert block_table.dim() == 2 and block_table.shape[0] == q.shape[0] == seq_lens.shape[0]
    assert k_pages.shape[3] == q.shape[2]


COMEM_PHASE_SPLIT = 1
COMEM_PHASE_COMBINE = 2


def comem_decode_attn_phases_async(q, k_pages, v_pages, block_table, seq_lens, softmax_scale: float, out,
                                   workspace, lse_out=None, stream=None,
                                   phases: int = COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE,
                                   grid_ctas=None, programmatic_launch=None, flags: int = 0) -> None:
    """Enqueue the selected kernels of one decode-attention step on ``stream``; returns at once."""
    _check_inputs(q, k_pages, v_pages, block_table, seq_lens)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    st = load_library().comem_decode_attn_phases_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), q.shape[1],
        k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream), int(phases),
        _opts(grid_ctas, programmatic_launch, flags))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn_phases_async")


def comem_decode_attn_async(q, k_pages, v_pages, block_table, seq_lens, softmax_scale: float, out,
                            workspace, lse_out=None, stream=None, grid_ctas=None, programmatic_launch=None, flags: int = 0) -> None:
    """Enqueue one decode-attention step (1 fused kernel launch) on ``stream``; returns at once."""
    _check_inputs(q, k_pages, v_pages, block_table, seq_lens)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    st = load_library().comem_decode_attn_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), q.shape[1],
        k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream), _opts(grid_ctas, programmatic_launch, flags))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn_async")


def comem_static_scratch_bytes() -> int:
    return int(load_library().comem_static_scratch_bytes())


def comem_decode_attn_static_async(q, k_pages, v_pages, block_table, seq_lens, softmax_scale: float, out,
                                   lse_out=None, stream=None, grid_ctas=None, programmatic_launch=None,
                                   flags: int = 0) -> None:
    """comem_decode_attn_async without a workspace: the scratch is a fixed device array inside the library (no
    allocation; shapes up to comem_static_scratch_bytes(); calls that overlap on the GPU race on it)."""
    _check_inputs(q, k_pages, v_pages, block_table, seq_lens)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    st = load_library().comem_decode_attn_static_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), q.shape[1],
        k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _stream(stream),
        _opts(grid_ctas, programmatic_launch, flags))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn_static_async")


def comem_decode_attn_window_async(q, k_pages, v_pages, block_table, seq_lens, softmax_scale: float, out,
                                   workspace, window: int, sink_tokens: int, lse_out=None, stream=None,
                                   grid_ctas=None, programmatic_launch=None, flags: int = 0) -> None:
    """Sliding-window + attention-sink decode attention (one fused launch on ``stream``)."""
    _check_inputs(q, k_pages, v_pages, block_table, seq_lens)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    st = load_library().comem_decode_attn_window_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), q.shape[1],
        k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream), int(window), int(sink_tokens),
        _opts(grid_ctas, programmatic_launch, flags))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn_window_async")


def comem_decode_attn_fp8_async(q, k_pages, v_pages, k_scale, v_scale, block_table, seq_lens,
                                softmax_scale: float, out, workspace, window: int = 0, sink_tokens: int = 0,
                                lse_out=None, stream=None, kv_layout: str = "NHD", grid_ctas=None,
                                programmatic_launch=None, flags: int = 0) -> None:
    """Decode attention over an FP8 (E4M3 bytes + fp32 page scales) KV cache; one fused launch.
    kv_layout "NHD": pools [P, page_size, Hkv, D]; "HND": pools [P, Hkv, page_size, D]."""
    assert kv_layout in ("NHD", "HND")
    hnd = kv_layout == "HND"
    assert q.is_cuda and q.dtype == torch.bfloat16 and q.is_contiguous() and q.dim() == 3
    for t in (k_pages, v_pages):
        assert t.is_cuda and t.dtype == torch.uint8 and t.is_contiguous() and t.dim() == 4
    assert k_pages.shape == v_pages.shape and k_pages.shape[3] == q.shape[2]
    page_size, hkv = (k_pages.shape[2], k_pages.shape[1]) if hnd else (k_pages.shape[1], k_pages.shape[2])
    for t in (k_scale, v_scale):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        assert tuple(t.shape) == (k_pages.shape[0], hkv)
    assert block_table.dtype == torch.int32 and block_table.is_contiguous() and block_table.shape[0] == q.shape[0]
    assert seq_lens.dtype == torch.int32 and seq_lens.is_contiguous() and seq_lens.shape == (q.shape[0],)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    st = load_library().comem_decode_attn_fp8_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(k_scale), _ptr(v_scale), _ptr(block_table), _ptr(seq_lens),
        q.shape[1], hkv, q.shape[2], page_size, ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream), int(window), int(sink_tokens), 1 if hnd else 0,
        _opts(grid_ctas, programmatic_launch, flags))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn_fp8_async")


def comem_decode_attn_offload_async(q, k_pages, v_pages, k_host, v_host, block_table, seq_lens, softmax_scale: float,
                                    out, workspace, lse_out=None, stream=None, grid_ctas=None,
                                    programmatic_launch=None, flags: int = 0) -> None:
    """Decode attention over a two-tier cache: block-table entries < 0 address pages of the pinned host pools
    (k_host, v_host: CPU tensors from .pin_memory()), entries >= 0 the device pools.  One fused launch."""
    _check_inputs(q, k_pages, v_pages, block_table, seq_lens)
    for t in (k_host, v_host):
        assert (not t.is_cuda) and t.is_pinned() and t.dtype == torch.bfloat16 and t.is_contiguous() and t.dim() == 4
        assert tuple(t.shape[1:]) == tuple(k_pages.shape[1:])
    assert k_host.shape == v_host.shape
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    st = load_library().comem_decode_attn_offload_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(k_host), _ptr(v_host), _ptr(block_table), _ptr(seq_lens),
        q.shape[1], k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], k_host.shape[0], _ptr(lse_out), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream), _opts(grid_ctas, programmatic_launch, flags))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn_offload_async")


def comem_pages_copy_async(k_src, v_src, k_dst, v_dst, src_ids, dst_ids, stream=None) -> None:
    """Copy pages src_ids[i] of (k_src, v_src) to pages dst_ids[i] of (k_dst, v_dst); pools are CUDA tensors or pinned
    CPU tensors of the same page shape; the id arrays are int32 CUDA tensors."""
    for t in (k_src, v_src, k_dst, v_dst):
        assert t.is_contiguous() and t.dim() == 4 and (t.is_cuda or t.is_pinned())
        assert tuple(t.shape[1:]) == tuple(k_src.shape[1:]) and t.dtype == k_src.dtype
    assert src_ids.is_cuda and dst_ids.is_cuda and src_ids.dtype == torch.int32 and dst_ids.dtype == torch.int32
    assert src_ids.is_contiguous() and dst_ids.is_contiguous() and src_ids.shape == dst_ids.shape and src_ids.dim() == 1
    page_bytes = k_src[0].numel() * k_src.element_size()
    st = load_library().comem_pages_copy_async(_ptr(k_src), _ptr(v_src), _ptr(k_dst), _ptr(v_dst), _ptr(src_ids),
                                               _ptr(dst_ids), src_ids.numel(), page_bytes, _stream(stream))
    if st != COMEM_OK:
        raise ComemError(st, "comem_pages_copy_async")


def comem_kv_append_fp8_async(k_pages, v_pages, k_scale, v_scale, block_table, seq_lens, new_k, new_v,
                              stream=None, kv_layout: str = "NHD") -> None:
    """Quantise one new bf16 (k, v) row per sequence into the E4M3 pools with the page's scales; seq_lens += 1."""
    assert kv_layout in ("NHD", "HND")
    hnd = kv_layout == "HND"
    assert k_pages.dtype == torch.uint8 and v_pages.dtype == torch.uint8 and k_pages.is_contiguous() and v_pages.is_contiguous()
    assert new_k.dtype == torch.bfloat16 and new_v.dtype == torch.bfloat16 and new_k.is_contiguous() and new_v.is_contiguous()
    page_size, hkv = (k_pages.shape[2], k_pages.shape[1]) if hnd else (k_pages.shape[1], k_pages.shape[2])
    assert tuple(new_k.shape) == (block_table.shape[0], hkv, k_pages.shape[3]) and new_v.shape == new_k.shape
    assert k_scale.dtype == torch.float32 and tuple(k_scale.shape) == (k_pages.shape[0], hkv) and v_scale.shape == k_scale.shape
    st = load_library().comem_kv_append_fp8_async(
        _ptr(k_pages), _ptr(v_pages), _ptr(k_scale), _ptr(v_scale), _ptr(block_table), _ptr(seq_lens), _ptr(new_k),
        _ptr(new_v), hkv, k_pages.shape[3], page_size, block_table.shape[0], block_table.shape[1], 1 if hnd else 0,
        _stream(stream))
    if st != COMEM_OK:
        raise ComemError(st, "comem_kv_append_fp8_async")


def comem_prefill_attn_async(q, k_pages, v_pages, block_table, seq_lens, q_start, softmax_scale: float, out,
                             lse_out=None, stream=None, programmatic_launch=None, grid_ctas=None) -> None:
    """Causal prefill attention of each sequence's last q_start[b+1] - q_start[b] tokens over the paged cache
    (one tcgen05 kernel on ``stream``).  q, out: bf16 [total_q, Hq, D]; q_start: int32 [batch + 1] on the device."""
    assert q.is_cuda and q.dtype == torch.bfloat16 and q.is_contiguous() and q.dim() == 3
    assert k_pages.dtype == torch.bfloat16 and v_pages.dtype == torch.bfloat16
    assert k_pages.is_contiguous() and v_pages.is_contiguous() and k_pages.dim() == 4 and k_pages.shape == v_pages.shape
    assert k_pages.shape[3] == q.shape[2]
    assert block_table.dtype == torch.int32 and block_table.is_contiguous() and block_table.dim() == 2
    assert seq_lens.dtype == torch.int32 and seq_lens.is_contiguous() and seq_lens.shape == (block_table.shape[0],)
    assert q_start.dtype == torch.int32 and q_start.is_contiguous() and q_start.shape == (block_table.shape[0] + 1,)
    assert out.dtype == torch.bfloat16 and out.shape == q.shape and out.is_contiguous()
    if lse_out is not None:
        assert lse_out.dtype == torch.float32 and lse_out.is_contiguous() and tuple(lse_out.shape) == tuple(q.shape[:2])
    st = load_library().comem_prefill_attn_async(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), _ptr(q_start), q.shape[1],
        k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        block_table.shape[0], q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _stream(stream),
        _opts(grid_ctas, programmatic_launch))
    if st != COMEM_OK:
        raise ComemError(st, "comem_prefill_attn_async")


def comem_decode_attn(q, k_pages, v_pages, block_table, seq_lens, softmax_scale: float, out=None,
                      workspace=None, lse_out=None):
    """Synchronous form (legacy default stream + cudaStreamSynchronize).  Returns ``out``."""
    _check_inputs(q, k_pages, v_pages, block_table, seq_lens)
    if out is None:
        out = torch.empty_like(q)
    if workspace is None:
        workspace = alloc_workspace(q, k_pages, block_table)
    torch.cuda.current_stream().synchronize()  # inputs were produced on torch's stream
    st = load_library().comem_decode_attn(
        _ptr(q), _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), q.shape[1],
        k_pages.shape[2], q.shape[2], k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out),
        q.shape[0], block_table.shape[1], k_pages.shape[0], _ptr(lse_out), _ptr(workspace),
        workspace.numel() * workspace.element_size())
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_attn")
    return out


def comem_validate_inputs(block_table, seq_lens, page_size: int, num_pages: int, workspace, stream=None) -> int:
    """Debug aid: COMEM_OK or COMEM_ERR_INVALID_ARG (returned, not raised) for the device-side data."""
    return int(load_library().comem_validate_inputs(
        _ptr(block_table), _ptr(seq_lens), block_table.shape[0], block_table.shape[1], int(page_size),
        int(num_pages), _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))


def comem_kv_append_async(k_pages, v_pages, block_table, seq_lens, new_k, new_v, stream=None) -> None:
    """Enqueue the KV append of one new (k, v) row per sequence; seq_lens += 1 on device."""
    assert new_k.dtype == torch.bfloat16 and new_v.dtype == torch.bfloat16
    assert new_k.is_contiguous() and new_v.is_contiguous() and new_k.shape == new_v.shape
    assert new_k.shape == (block_table.shape[0], k_pages.shape[2], k_pages.shape[3])
    st = load_library().comem_kv_append_async(
        _ptr(k_pages), _ptr(v_pages), _ptr(block_table), _ptr(seq_lens), _ptr(new_k), _ptr(new_v),
        k_pages.shape[2], k_pages.shape[3], k_pages.shape[1], block_table.shape[0],
        block_table.shape[1], _stream(stream))
    if st != COMEM_OK:
        raise ComemError(st, "comem_kv_append_async")


def comem_decode_step_host(q_host, new_k_host, new_v_host, k_pages, v_pages, block_table, seq_lens,
                           softmax_scale: float, out_host, workspace, lse_host=None, stream=None) -> None:
    """One whole decode step from HOST q / new k / new v rows to a HOST output (synchronous)."""
    assert q_host.device.type == "cpu" and out_host.device.type == "cpu"
    assert q_host.dtype == torch.bfloat16 and out_host.dtype == torch.bfloat16
    assert q_host.is_contiguous() and out_host.is_contiguous() and out_host.shape == q_host.shape
    st = load_library().comem_decode_step_host(
        _ptr(q_host), _ptr(new_k_host), _ptr(new_v_host), _ptr(k_pages), _ptr(v_pages),
        _ptr(block_table), _ptr(seq_lens), q_host.shape[1], k_pages.shape[2], q_host.shape[2],
        k_pages.shape[1], ctypes.c_float(softmax_scale), _ptr(out_host), q_host.shape[0],
        block_table.shape[1], k_pages.shape[0], _ptr(lse_host), _ptr(workspace),
        workspace.numel() * workspace.element_size(), _stream(stream))
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_step_host")


class DecodeStepHost:
    """comem_decode_step_host with the arguments marshalled ONCE: a serving loop calls the same step on the same
    buffers thousands of times, and building twenty ctypes arguments from torch tensors costs more host time than the
    GPU needs for a 32K-token step.  ``step = DecodeStepHost(...)`` checks and converts everything, ``step()`` is one
    foreign call.  The tensors must stay alive and in place; ``rebind(q_host=..., new_k_host=..., new_v_host=...,
    out_host=...)`` swaps host buffers (e.g. a ring of pinned rows) without re-marshalling the rest."""

    def __init__(self, q_host, new_k_host, new_v_host, k_pages, v_pages, block_table, seq_lens, softmax_scale: float,
                 out_host, workspace, lse_host=None, stream=None):
        assert q_host.device.type == "cpu" and out_host.device.type == "cpu"
        assert q_host.dtype == torch.bfloat16 and out_host.dtype == torch.bfloat16
        assert q_host.is_contiguous() and out_host.is_contiguous() and out_host.shape == q_host.shape
        self._fn = load_library().comem_decode_step_host
        self._keep = (q_host, new_k_host, new_v_host, k_pages, v_pages, block_table, seq_lens, out_host, workspace, lse_host)
        self._args = [_ptr(q_host), _ptr(new_k_host), _ptr(new_v_host), _ptr(k_pages), _ptr(v_pages), _ptr(block_table),
                      _ptr(seq_lens), q_host.shape[1], k_pages.shape[2], q_host.shape[2], k_pages.shape[1],
                      ctypes.c_float(softmax_scale), _ptr(out_host), q_host.shape[0], block_table.shape[1],
                      k_pages.shape[0], _ptr(lse_host), _ptr(workspace), workspace.numel() * workspace.element_size(),
                      _stream(stream)]

    def rebind(self, q_host=None, new_k_host=None, new_v_host=None, out_host=None):
        for i, t in ((0, q_host), (1, new_k_host), (2, new_v_host), (12, out_host)):
            if t is not None:
                assert t.device.type == "cpu" and t.is_contiguous()
                self._args[i] = _ptr(t)
        self._keep = self._keep + (q_host, new_k_host, new_v_host, out_host)
        return self

    def __call__(self) -> None:
        st = self._fn(*self._args)
        if st != COMEM_OK:
            raise ComemError(st, "comem_decode_step_host")


def comem_decode_step_host_fp8(q_host, new_k_host, new_v_host, k_pages, v_pages, k_scale, v_scale, block_table, seq_lens,
                               softmax_scale: float, out_host, workspace, lse_host=None, stream=None,
                               kv_layout: str = "NHD") -> None:
    """comem_decode_step_host for the FP8 cache: host q / new k / new v rows in (bf16), quantising append, FP8 decode
    attention, host out back (synchronous)."""
    assert kv_layout in ("NHD", "HND")
    hnd = kv_layout == "HND"
    assert q_host.device.type == "cpu" and out_host.device.type == "cpu"
    assert q_host.dtype == torch.bfloat16 and out_host.dtype == torch.bfloat16 and k_pages.dtype == torch.uint8
    assert q_host.is_contiguous() and out_host.is_contiguous() and out_host.shape == q_host.shape
    page_size, hkv = (k_pages.shape[2], k_pages.shape[1]) if hnd else (k_pages.shape[1], k_pages.shape[2])
    st = load_library().comem_decode_step_host_fp8(
        _ptr(q_host), _ptr(new_k_host), _ptr(new_v_host), _ptr(k_pages), _ptr(v_pages), _ptr(k_scale), _ptr(v_scale),
        _ptr(block_table), _ptr(seq_lens), q_host.shape[1], hkv, q_host.shape[2], page_size,
        ctypes.c_float(softmax_scale), _ptr(out_host), q_host.shape[0], block_table.shape[1], k_pages.shape[0],
        _ptr(lse_host), _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream), 1 if hnd else 0)
    if st != COMEM_OK:
        raise ComemError(st, "comem_decode_step_host_fp8")
