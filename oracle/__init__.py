"""oracle/ — TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front-end for ``decode_attn_oracle.c`` (plain fp64 CPU paged decode
attention; see that file's header for the paper citations and the pins).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2605_30842_b200`` and the CUDA path imports nothing from here.

Argument marshalling only: every array is handed to C as raw bits (bf16 as
uint16); all arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "decode_attn_oracle.c")
_LIB = os.path.join(_HERE, "libdecode_attn_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, no fast-math, OpenMP over rows)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        c = ctypes
        vp, i32, i64, f32 = c.c_void_p, c.c_int, c.c_int64, c.c_float
        lib.oracle_decode_attn.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, vp,
                                           i32, i32, vp, i64, i32]
        lib.oracle_decode_attn.restype = i32
        lib.oracle_decode_attn_window.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, i32, i32, vp, vp,
                                                  i32, i32, i32]
        lib.oracle_decode_attn_window.restype = i32
        lib.oracle_decode_attn_fp8.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, i32, i32, i32, vp, vp,
                                               i32, i32, i32]
        lib.oracle_decode_attn_fp8.restype = i32
        lib.oracle_e4m3_decode.argtypes = [i32]
        lib.oracle_e4m3_decode.restype = c.c_double
        lib.oracle_decode_attn_partial.argtypes = [vp, vp, vp, vp, vp, i32, i32, i32, i32, f32,
                                                   i32, i32, i64, i64, i32, vp, vp, vp]
        lib.oracle_decode_attn_partial.restype = i32
        lib.oracle_lse_merge.argtypes = [vp, vp, vp, i32, i32, vp, vp]
        lib.oracle_lse_merge.restype = i32
        lib.oracle_kv_append.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32]
        lib.oracle_kv_append.restype = i32
        lib.oracle_e4m3_encode.argtypes = [f32]
        lib.oracle_e4m3_encode.restype = i32
        lib.oracle_kv_append_fp8.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32]
        lib.oracle_kv_append_fp8.restype = i32
        lib.oracle_prefill_attn.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, f32, vp, vp, i32, i32, i32]
        lib.oracle_prefill_attn.restype = i32
        lib.oracle_max_threads.restype = i32
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def as_bits(x) -> np.ndarray:
    """torch bf16 CPU tensor or numpy uint16 array -> C-contiguous numpy uint16 (raw bits)."""
    if isinstance(x, np.ndarray):
        assert x.dtype == np.uint16, x.dtype
        return np.ascontiguousarray(x)
    import torch  # plumbing only

    assert x.dtype == torch.bfloat16 and x.device.type == "cpu", (x.dtype, x.device)
    return np.ascontiguousarray(x.contiguous().view(torch.int16).numpy().view(np.uint16))


def _as_i32(x) -> np.ndarray:
    if not isinstance(x, np.ndarray):
        x = x.cpu().numpy()
    return np.ascontiguousarray(x.astype(np.int32, copy=False))


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _dims(q, k_pages, block_table):
    batch, hq, d = q.shape
    p, ps, hkv, d2 = k_pages.shape
    assert d2 == d and block_table.shape[0] == batch
    return batch, hq, hkv, d, ps, block_table.shape[1], p


def decode_attn(q, k_pages, v_pages, block_table, seq_lens, softmax_scale, pairs=None,
                num_threads: int = 0):
    """fp64 paged decode attention.  Returns (out, lse) as numpy float64.

    out is [batch, Hq, D] (or [num_pairs, D] when ``pairs`` — an int array of
    (b, h) rows — is given); lse is [batch, Hq] (or [num_pairs]).
    """
    lib = _load()
    qb, kb, vb = as_bits(q), as_bits(k_pages), as_bits(v_pages)
    bt, sl = _as_i32(block_table), _as_i32(seq_lens)
    batch, hq, hkv, d, ps, maxp, _ = _dims(qb, kb, bt)
    assert vb.shape == kb.shape and sl.shape == (batch,)
    scale = np.float32(softmax_scale)
    if pairs is None:
        out = np.empty((batch, hq, d), np.float64)
        lse = np.empty((batch, hq), np.float64)
        pr, npairs = None, 0
    else:
        pr = np.ascontiguousarray(np.asarray(pairs, np.int32).reshape(-1, 2))
        npairs = pr.shape[0]
        out = np.empty((npairs, d), np.float64)
        lse = np.empty((npairs,), np.float64)
    rc = lib.oracle_decode_attn(_p(qb), _p(kb), _p(vb), _p(bt), _p(sl), hq, hkv, d, ps,
                                ctypes.c_float(float(scale)), _p(out), _p(lse), batch, maxp,
                                _p(pr), npairs, int(num_threads))
    if rc != 0:
        raise ValueError(f"oracle_decode_attn: invalid argument (rc={rc})")
    return out, lse


def decode_attn_window(q, k_pages, v_pages, block_table, seq_lens, softmax_scale, window: int,
                       sink_tokens: int, num_threads: int = 0):
    """Sliding-window + attention-sink variant: the query (position L-1) attends t < sink_tokens or
    t >= L - window.  Returns (out [batch, Hq, D], lse [batch, Hq]) as numpy float64."""
    lib = _load()
    qb, kb, vb = as_bits(q), as_bits(k_pages), as_bits(v_pages)
    bt, sl = _as_i32(block_table), _as_i32(seq_lens)
    batch, hq, hkv, d, ps, maxp, _ = _dims(qb, kb, bt)
    out = np.empty((batch, hq, d), np.float64)
    lse = np.empty((batch, hq), np.float64)
    rc = lib.oracle_decode_attn_window(_p(qb), _p(kb), _p(vb), _p(bt), _p(sl), hq, hkv, d, ps,
                                       ctypes.c_float(float(np.float32(softmax_scale))), int(window),
                                       int(sink_tokens), _p(out), _p(lse), batch, maxp, int(num_threads))
    if rc != 0:
        raise ValueError(f"oracle_decode_attn_window: invalid argument (rc={rc})")
    return out, lse


def _as_u8(x) -> np.ndarray:
    """torch uint8 / float8_e4m3fn CPU tensor or numpy uint8 array -> C-contiguous numpy uint8 (raw bytes)."""
    if isinstance(x, np.ndarray):
        assert x.dtype == np.uint8, x.dtype
        return np.ascontiguousarray(x)
    import torch  # plumbing only

    assert x.device.type == "cpu" and x.element_size() == 1, (x.dtype, x.device)
    return np.ascontiguousarray(x.contiguous().view(torch.uint8).numpy())


def e4m3_decode(byte: int) -> float:
    """Value of one OCP FP8 E4M3 byte as the oracle reads it (NaN for 0x7f / 0xff)."""
    return float(_load().oracle_e4m3_decode(int(byte)))


def decode_attn_fp8(q, k_pages, v_pages, k_scale, v_scale, block_table, seq_lens, softmax_scale,
                    window: int = 0, sink_tokens: int = 0, num_threads: int = 0, kv_layout: str = "NHD"):
    """FP8 (E4M3 + one fp32 scale per physical page and kv head) KV-cache variant, reading R18.
    k_pages / v_pages: raw bytes [P, page_size, Hkv, D] (kv_layout "NHD") or [P, Hkv, page_size, D] ("HND");
    k_scale / v_scale: fp32 [P, Hkv].
    Returns (out [batch, Hq, D], lse [batch, Hq]) as numpy float64."""
    lib = _load()
    qb, kb, vb = as_bits(q), _as_u8(k_pages), _as_u8(v_pages)
    bt, sl = _as_i32(block_table), _as_i32(seq_lens)
    assert kv_layout in ("NHD", "HND")
    batch, hq, hkv, d, ps, maxp, npages = _dims(qb, kb, bt)
    if kv_layout == "HND":
        hkv, ps = ps, hkv
    ks = np.ascontiguousarray(np.asarray(k_scale.cpu().numpy() if hasattr(k_scale, "cpu") else k_scale, np.float32))
    vs = np.ascontiguousarray(np.asarray(v_scale.cpu().numpy() if hasattr(v_scale, "cpu") else v_scale, np.float32))
    assert vb.shape == kb.shape and ks.shape == (npages, hkv) and vs.shape == (npages, hkv)
    out = np.empty((batch, hq, d), np.float64)
    lse = np.empty((batch, hq), np.float64)
    rc = lib.oracle_decode_attn_fp8(_p(qb), _p(kb), _p(vb), _p(ks), _p(vs), _p(bt), _p(sl), hq, hkv, d, ps,
                                    ctypes.c_float(float(np.float32(softmax_scale))), int(window),
                                    int(sink_tokens), 1 if kv_layout == "HND" else 0, _p(out), _p(lse), batch, maxp,
                                    int(num_threads))
    if rc != 0:
        raise ValueError(f"oracle_decode_attn_fp8: invalid argument (rc={rc})")
    return out, lse


def decode_attn_partial(q, k_pages, v_pages, block_table, seq_lens, softmax_scale, b, h, t0, t1):
    """Un-normalised (acc[D], m, l) of row (b, h) over tokens [t0, t1)."""
    lib = _load()
    qb, kb, vb = as_bits(q), as_bits(k_pages), as_bits(v_pages)
    bt, sl = _as_i32(block_table), _as_i32(seq_lens)
    batch, hq, hkv, d, ps, maxp, _ = _dims(qb, kb, bt)
    acc = np.empty((d,), np.float64)
    m = np.empty((1,), np.float64)
    l = np.empty((1,), np.float64)
    rc = lib.oracle_decode_attn_partial(_p(qb), _p(kb), _p(vb), _p(bt), _p(sl), hq, hkv, d, ps,
                                        ctypes.c_float(float(np.float32(softmax_scale))), int(b),
                                        int(h), int(t0), int(t1), maxp, _p(acc), _p(m), _p(l))
    if rc != 0:
        raise ValueError("oracle_decode_attn_partial: invalid argument")
    return acc, float(m[0]), float(l[0])


def lse_merge(acc, m, l):
    """Combine S partials of one row: acc [S, D], m [S], l [S] -> (out [D], lse)."""
    lib = _load()
    acc = np.ascontiguousarray(acc, np.float64)
    m = np.ascontiguousarray(m, np.float64)
    l = np.ascontiguousarray(l, np.float64)
    s, d = acc.shape
    out = np.empty((d,), np.float64)
    lse = np.empty((1,), np.float64)
    lib.oracle_lse_merge(_p(acc), _p(m), _p(l), s, d, _p(out), _p(lse))
    return out, float(lse[0])


def kv_append(k_bits, v_bits, block_table, seq_lens, new_k, new_v):
    """In place: append one (k, v) row per sequence, seq_lens += 1.

    k_bits / v_bits / seq_lens must be writable C-contiguous numpy arrays
    (uint16, uint16, int32); new_k / new_v are bf16 [batch, Hkv, D].
    """
    lib = _load()
    assert k_bits.dtype == np.uint16 and k_bits.flags.c_contiguous and k_bits.flags.writeable
    assert v_bits.dtype == np.uint16 and v_bits.flags.c_contiguous and v_bits.flags.writeable
    assert seq_lens.dtype == np.int32 and seq_lens.flags.c_contiguous
    bt = _as_i32(block_table)
    nk, nv = as_bits(new_k), as_bits(new_v)
    _, ps, hkv, d = k_bits.shape
    rc = lib.oracle_kv_append(_p(k_bits), _p(v_bits), _p(bt), _p(seq_lens), _p(nk), _p(nv), hkv,
                              d, ps, bt.shape[0], bt.shape[1])
    if rc != 0:
        raise ValueError("oracle_kv_append: sequence would outgrow its block-table row")


def e4m3_encode(x: float) -> int:
    """fp32 -> E4M3 byte, round-to-nearest-even, saturating at +-448 (NaN -> 0x7f)."""
    return int(_load().oracle_e4m3_encode(ctypes.c_float(x)))


def kv_append_fp8(k_bytes, v_bytes, k_scale, v_scale, block_table, seq_lens, new_k, new_v, kv_layout: str = "NHD"):
    """In place: quantise one new bf16 (k, v) row per sequence with its page's scales into the E4M3 pools
    (numpy uint8, writable, C-contiguous), seq_lens (numpy int32) += 1."""
    lib = _load()
    assert k_bytes.dtype == np.uint8 and k_bytes.flags.c_contiguous and k_bytes.flags.writeable
    assert v_bytes.dtype == np.uint8 and v_bytes.flags.c_contiguous and v_bytes.flags.writeable
    assert seq_lens.dtype == np.int32 and seq_lens.flags.c_contiguous
    ks = np.ascontiguousarray(np.asarray(k_scale, np.float32))
    vs = np.ascontiguousarray(np.asarray(v_scale, np.float32))
    bt = _as_i32(block_table)
    nk, nv = as_bits(new_k), as_bits(new_v)
    hnd = kv_layout == "HND"
    _, a, b_, d = k_bytes.shape
    hkv, ps = (a, b_) if hnd else (b_, a)
    rc = lib.oracle_kv_append_fp8(_p(k_bytes), _p(v_bytes), _p(ks), _p(vs), _p(bt), _p(seq_lens), _p(nk), _p(nv),
                                  hkv, d, ps, bt.shape[0], bt.shape[1], 1 if hnd else 0)
    if rc != 0:
        raise ValueError("oracle_kv_append_fp8: sequence would outgrow its block-table row")


def prefill_attn(q, k_pages, v_pages, block_table, seq_lens, q_start, softmax_scale, num_threads: int = 0):
    """Causal prefill attention of the last q_len_b = q_start[b+1] - q_start[b] tokens of every sequence over the
    paged cache (reading R20).  q: bf16 [total_q, Hq, D] ragged.  Returns (out [total_q, Hq, D], lse [total_q, Hq])."""
    lib = _load()
    qb, kb, vb = as_bits(q), as_bits(k_pages), as_bits(v_pages)
    bt, sl, qs = _as_i32(block_table), _as_i32(seq_lens), _as_i32(q_start)
    total_q, hq, d = qb.shape
    _, ps, hkv, _ = kb.shape
    batch = sl.shape[0]
    assert qs.shape == (batch + 1,) and int(qs[-1]) == total_q
    out = np.empty((total_q, hq, d), np.float64)
    lse = np.empty((total_q, hq), np.float64)
    rc = lib.oracle_prefill_attn(_p(qb), _p(kb), _p(vb), _p(bt), _p(sl), _p(qs), hq, hkv, d, ps,
                                 ctypes.c_float(float(np.float32(softmax_scale))), _p(out), _p(lse), batch,
                                 bt.shape[1], int(num_threads))
    if rc != 0:
        raise ValueError("oracle_prefill_attn: invalid argument")
    return out, lse
