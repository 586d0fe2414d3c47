"""CPU-side checks of the C-ABI library: it loads without a GPU, exports every symbol
include/comem_decode_attn.h declares, validates arguments, and its host scheduler mirror
partitions the tile space exactly.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2605_30842_b200 as comem

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "comem_decode_attn.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2605_30842_b200 import build

    build.build()
    return comem.load_library()


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(comem_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_all_exported(lib):
    names = declared_symbols()
    assert {"comem_decode_attn", "comem_decode_attn_async", "comem_decode_attn_workspace_bytes",
            "comem_kv_append_async", "comem_decode_step_host", "comem_schedule_host",
            "comem_status_string", "comem_version"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in the header but not exported"


def test_version_and_status_strings(lib):
    assert comem.comem_version() >= 100
    seen = {comem.comem_status_string(s) for s in range(5)}
    assert len(seen) == 5 and "ok" in seen
    assert comem.comem_status_string(99) == "unknown status"


def test_workspace_bytes_pure_host(lib):
    a = comem.comem_decode_attn_workspace_bytes(1, 64, 8, 128, 16, 2048)
    b = comem.comem_decode_attn_workspace_bytes(32, 64, 8, 128, 16, 4096)
    assert 0 < a < b < 64 << 20 and a % 256 == 0
    assert comem.comem_decode_attn_workspace_bytes(0, 64, 8, 128, 16, 1) == 0


def _call(lib, **over):
    """comem_decode_attn_async with dummy non-null pointers; validation must reject before any launch."""
    a = dict(q=256, k=256, v=512, bt=256, sl=256, hq=64, hkv=8, d=128, ps=16, scale=0.1, out=256,
             batch=1, maxp=16, npages=16, lse=None, ws=256, wsb=1 << 26, stream=None)
    a.update(over)
    return lib.comem_decode_attn_async(a["q"], a["k"], a["v"], a["bt"], a["sl"], a["hq"], a["hkv"],
                                       a["d"], a["ps"], ctypes.c_float(a["scale"]), a["out"],
                                       a["batch"], a["maxp"], a["npages"], a["lse"], a["ws"], a["wsb"],
                                       a["stream"], None)


def test_argument_validation(lib):
    assert _call(lib, q=None) == comem.COMEM_ERR_INVALID_ARG
    assert _call(lib, out=None) == comem.COMEM_ERR_INVALID_ARG
    assert _call(lib, batch=0) == comem.COMEM_ERR_INVALID_ARG
    assert _call(lib, hq=60) == comem.COMEM_ERR_INVALID_ARG            # 60 % 8 != 0
    assert _call(lib, scale=float("nan")) == comem.COMEM_ERR_INVALID_ARG
    assert _call(lib, scale=-1.0) == comem.COMEM_ERR_INVALID_ARG
    assert _call(lib, q=258) == comem.COMEM_ERR_INVALID_ARG            # misaligned
    assert _call(lib, d=96) == comem.COMEM_ERR_UNSUPPORTED
    assert _call(lib, ps=8) == comem.COMEM_ERR_UNSUPPORTED
    assert _call(lib, hq=128) == comem.COMEM_ERR_UNSUPPORTED           # group 16
    assert _call(lib, batch=5000) == comem.COMEM_ERR_UNSUPPORTED
    assert _call(lib, npages=1 << 28) == comem.COMEM_ERR_UNSUPPORTED   # row coordinate overflows int32
    assert _call(lib, ws=None) == comem.COMEM_ERR_WORKSPACE
    assert _call(lib, wsb=1024) == comem.COMEM_ERR_WORKSPACE
    # fully valid arguments but no usable device here -> CUDA error, never a crash or a CPU fallback
    import torch
    if not torch.cuda.is_available():
        assert _call(lib) in (comem.COMEM_ERR_CUDA, comem.COMEM_ERR_UNSUPPORTED)


def test_missing_library_fails_loudly(monkeypatch):
    from paper_2605_30842_b200 import binding

    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", "/nonexistent/libcomem_decode.so")
    with pytest.raises(RuntimeError, match="no CPU or PyTorch fallback"):
        binding.load_library()


@pytest.mark.parametrize("lens,hkv,grid", [([32768], 8, 296), ([512], 1, 296), ([1], 1, 296),
                                            ([0, 0], 2, 8), ([100, 0, 37, 5000, 16], 8, 296),
                                            (list(range(1, 200)), 4, 296)])
def test_schedule_partitions_tile_space(lib, lens, hkv, grid):
    begins = comem.comem_schedule_host(lens, hkv, grid)
    tiles = sum((l + 15) // 16 for l in lens) * hkv
    if tiles == 0:
        assert begins == [0]
        return
    assert begins[0] == 0 and begins[-1] == tiles
    sizes = np.diff(begins)
    assert (sizes >= 0).all() and sizes.max() - sizes.min() <= 1       # balanced to one tile
    nc = len(begins) - 1
    assert nc == min(grid, max(1, -(-tiles // 16)))    # schedule.cuh kMinTilesPerCta = 16


def test_schedule_segment_aligned_variant(lib):
    """Few long segments (C2: 8 segments of 2048 tiles on 148 CTAs): whole CTAs are dealt to segments,
    so no CTA straddles a segment boundary, at the price of 18 vs 19 CTAs per segment; many
    segments (C3-like) keep the linear cut, balanced to one tile."""
    begins = comem.comem_schedule_host([32768], 8, 148)
    assert len(begins) == 149 and begins[0] == 0 and begins[-1] == 8 * 2048
    sizes = np.diff(begins)
    assert sizes.min() >= 107 and sizes.max() <= 114
    for i in range(148):
        assert begins[i] // 2048 == (begins[i + 1] - 1) // 2048, i      # one segment per CTA
    per_seg = np.bincount(np.asarray(begins[:-1]) // 2048, minlength=8)
    assert sorted(set(per_seg.tolist())) == [18, 19] and per_seg.sum() == 148
    # the price is capped: 2 sequences x 8 heads of 65536 tokens would cost 12 tiles -> linear cut
    begins = comem.comem_schedule_host([65536, 65536], 8, 148)
    sizes = np.diff(begins)
    assert sizes.max() - sizes.min() <= 1
    # more segments than kAlignedMaxSegs -> linear cut
    begins = comem.comem_schedule_host([20000] * 32, 8, 148)
    sizes = np.diff(begins)
    assert sizes.max() - sizes.min() <= 1


def test_fp8_entry_point_validates_before_any_launch(lib):
    """comem_decode_attn_fp8_async: null scales, an unsupported head_dim and an unknown layout are rejected on the host."""
    import ctypes
    vp = ctypes.c_void_p
    d = vp(0x1000)

    def call(ks=d, vs=d, head_dim=128, layout=0, sinks=0):
        return lib.comem_decode_attn_fp8_async(d, d, d, ks, vs, d, d, 64, 8, head_dim, 16, ctypes.c_float(0.088), d, 1,
                                               2048, 4096, None, d, 1 << 30, None, 0, sinks, layout, None)

    assert call(ks=None) == comem.COMEM_ERR_INVALID_ARG
    assert call(vs=None) == comem.COMEM_ERR_INVALID_ARG
    assert call(head_dim=96) == comem.COMEM_ERR_UNSUPPORTED
    assert call(layout=7) == comem.COMEM_ERR_INVALID_ARG
    assert call(sinks=-1) == comem.COMEM_ERR_INVALID_ARG
    # valid arguments get as far as the device check; only where there is no GPU: with one, these made-up pointers would
    # reach a launch
    import torch
    if not torch.cuda.is_available():
        assert call() in (comem.COMEM_ERR_CUDA, comem.COMEM_ERR_UNSUPPORTED, comem.COMEM_ERR_WORKSPACE)


def test_round2_entry_points_validate_arguments_on_the_host(lib):
    """Host-side validation of the round-2 calls (no device work is reached): null pointers, bad sizes, unknown launch
    flags.  Each returns a status code; none crashes, none falls back to a CPU path."""
    import ctypes as C
    vp = C.c_void_p
    lib.comem_pages_copy_async.argtypes = [vp, vp, vp, vp, vp, vp, C.c_int, C.c_size_t, vp]
    lib.comem_pages_copy_async.restype = C.c_int
    buf = (C.c_char * 4096)()
    p = C.cast(buf, vp)
    assert lib.comem_pages_copy_async(None, p, p, p, p, p, 1, 4096, None) == comem.COMEM_ERR_INVALID_ARG
    assert lib.comem_pages_copy_async(p, p, p, p, p, p, 1, 100, None) == comem.COMEM_ERR_INVALID_ARG      # not a multiple of 16
    assert lib.comem_pages_copy_async(p, p, p, p, p, p, -1, 4096, None) == comem.COMEM_ERR_INVALID_ARG
    lib.comem_decode_attn_offload_async.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_float,
                                                    vp, C.c_int, C.c_int, C.c_int64, C.c_int64, vp, vp, C.c_size_t, vp, vp]
    lib.comem_decode_attn_offload_async.restype = C.c_int
    assert lib.comem_decode_attn_offload_async(p, p, p, None, p, p, p, 8, 2, 128, 16, C.c_float(0.1), p, 1, 4, 8, 8, None, p,
                                               1 << 30, None, None) == comem.COMEM_ERR_INVALID_ARG       # no host K pool
    # unknown launch flag bits are rejected before anything is launched
    opts = comem.LaunchOpts(0, -1, 1 << 10)
    lib.comem_decode_attn_async.restype = C.c_int
    st = lib.comem_decode_attn_async(p, p, p, p, p, 8, 2, 128, 16, C.c_float(0.1), p, 1, 4, 8, None, p,
                                     comem.comem_decode_attn_workspace_bytes(1, 8, 2, 128, 16, 4), None, C.byref(opts))
    assert st == comem.COMEM_ERR_INVALID_ARG     # whatever the alignment of `buf` happens to be
    # the Algorithm-1 step scheduler: null model / event, bad token counts
    ev = comem.KstepEvent(1, 0, 0, 1, 0, 0)
    m = comem.KstepModel()
    lib.comem_kstep_step_async.restype = C.c_int
    assert lib.comem_kstep_step_async(None, 64, 32, 1, 0, C.byref(m), None, None, None, None, None, None) == comem.COMEM_ERR_INVALID_ARG
    assert lib.comem_kstep_step_async(C.byref(ev), 64, 32, 1, 0, C.byref(m), None, None, None, None, None, None) == comem.COMEM_ERR_INVALID_ARG
    lib.comem_decode_step_host_fp8.restype = C.c_int
    assert lib.comem_decode_step_host_fp8(None, p, p, p, p, p, p, p, p, 8, 2, 128, 16, C.c_float(0.1), p, 1, 4, 8, None, p, 1 << 20,
                                          None, 0) == comem.COMEM_ERR_INVALID_ARG
