"""Seeded synthetic inputs for the paged decode-attention path.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.
It holds none of the method's arithmetic (no dot products, no softmax, no
combine): it only draws random tensors, deals physical pages and writes the
block table.  torch is used as the random source and container.

The five named workloads are BASELINE.json's ``configs`` made concrete
(DESIGN.md "Input recipe").  They stand in for the paper's
measurements on SWE-Bench-Verified trajectories and on "random data with fixed
lengths and a constant batch size": model geometries 64q/8kv/128
(one layer of the 32B agent) and 32q/8kv/128 (one layer of the 4B memory model,
PAPER.md L49), agent prompt lengths 30-46K, memory inputs up
to 128K, 64-step trajectories.

Values come from ``torch.Generator(device).manual_seed(seed)``; the CPU and CUDA
generators give different streams, so a workload is identified by (name, seed,
device).  Whatever is generated, the SAME BITS go to the oracle and to the GPU
path (copy, never regenerate).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np
import torch


@dataclasses.dataclass
class DecodeBatch:
    """One decode step's inputs, in the C-ABI's layouts (include/comem_decode_attn.h)."""

    q: torch.Tensor            # bf16 [batch, Hq, D]
    k_pages: torch.Tensor      # bf16 [P, page_size, Hkv, D]
    v_pages: torch.Tensor      # bf16 [P, page_size, Hkv, D]
    block_table: torch.Tensor  # int32 [batch, max_pages_per_seq]
    seq_lens: torch.Tensor     # int32 [batch]
    softmax_scale: float       # the fp32 value handed to the ABI
    name: str = ""
    seed: int = 0

    @property
    def batch(self) -> int:
        return self.q.shape[0]

    @property
    def num_q_heads(self) -> int:
        return self.q.shape[1]

    @property
    def num_kv_heads(self) -> int:
        return self.k_pages.shape[2]

    @property
    def head_dim(self) -> int:
        return self.q.shape[2]

    @property
    def page_size(self) -> int:
        return self.k_pages.shape[1]

    @property
    def num_pages(self) -> int:
        return self.k_pages.shape[0]

    @property
    def max_pages_per_seq(self) -> int:
        return self.block_table.shape[1]

    def algorithmic_bytes(self) -> int:
        """KV + Q bytes one decode step must read:
        sum_b L_b * Hkv * D * 2 (K and V) * 2 B  +  B * Hq * D * 2 B."""
        tokens = int(self.seq_lens.to(torch.int64).sum().item())
        kv = tokens * self.num_kv_heads * self.head_dim * 2 * 2
        qb = self.batch * self.num_q_heads * self.head_dim * 2
        return kv + qb

    def to(self, device) -> "DecodeBatch":
        return dataclasses.replace(
            self, q=self.q.to(device), k_pages=self.k_pages.to(device),
            v_pages=self.v_pages.to(device), block_table=self.block_table.to(device),
            seq_lens=self.seq_lens.to(device))

    def checksums(self) -> dict:
        """xor/sum of the raw bits, so two runs can be told to have had the same inputs."""
        def cs(t: torch.Tensor) -> int:
            bits = t.contiguous().view(torch.int16) if t.dtype == torch.bfloat16 else t
            return int(bits.to(torch.int64).sum().item())
        return {"q": cs(self.q), "block_table": cs(self.block_table), "seq_lens": cs(self.seq_lens)}


@dataclasses.dataclass
class Fp8DecodeBatch:
    """A decode batch whose KV cache is stored as FP8 E4M3 bytes with one fp32 scale per
    (physical page, kv head) and per pool (reading R18)."""

    q: torch.Tensor            # bf16 [batch, Hq, D]
    k_pages: torch.Tensor      # uint8 (E4M3 bytes) [P, page_size, Hkv, D]
    v_pages: torch.Tensor      # uint8 (E4M3 bytes) [P, page_size, Hkv, D]
    k_scale: torch.Tensor      # fp32 [P, Hkv]
    v_scale: torch.Tensor      # fp32 [P, Hkv]
    block_table: torch.Tensor  # int32 [batch, max_pages_per_seq]
    seq_lens: torch.Tensor     # int32 [batch]
    softmax_scale: float
    name: str = ""
    seed: int = 0
    kv_layout: str = "NHD"     # "HND": k_pages / v_pages are [P, Hkv, page_size, D]

    batch = property(lambda self: self.q.shape[0])
    num_q_heads = property(lambda self: self.q.shape[1])
    num_kv_heads = property(lambda self: self.k_pages.shape[1 if self.kv_layout == "HND" else 2])
    head_dim = property(lambda self: self.q.shape[2])
    page_size = property(lambda self: self.k_pages.shape[2 if self.kv_layout == "HND" else 1])
    num_pages = property(lambda self: self.k_pages.shape[0])
    max_pages_per_seq = property(lambda self: self.block_table.shape[1])

    def algorithmic_bytes(self, kept_tokens: Optional[int] = None) -> int:
        """K and V bytes (1 B per element) of the tokens read, their page scales (2 x 4 B per page and
        kv head) and Q."""
        ps = self.page_size
        lens = self.seq_lens.to(torch.int64)
        tokens = int(lens.sum().item()) if kept_tokens is None else int(kept_tokens)
        pages = int(((lens + ps - 1) // ps).sum().item()) if kept_tokens is None else (int(kept_tokens) + ps - 1) // ps
        return (tokens * self.num_kv_heads * self.head_dim * 2 + pages * self.num_kv_heads * 8 +
                self.batch * self.num_q_heads * self.head_dim * 2)

    def to(self, device) -> "Fp8DecodeBatch":
        mv = lambda t: t.to(device)
        return dataclasses.replace(self, q=mv(self.q), k_pages=mv(self.k_pages), v_pages=mv(self.v_pages),
                                   k_scale=mv(self.k_scale), v_scale=mv(self.v_scale),
                                   block_table=mv(self.block_table), seq_lens=mv(self.seq_lens))


E4M3_MAX = 448.0


def _quantize_pool_e4m3(pages: torch.Tensor, chunk_pages: int = 4096):
    """[P, ps, Hkv, D] bf16 -> (uint8 E4M3 bytes, fp32 scale [P, Hkv]).  Input recipe, not the method:
    scale = amax over the (page, kv head) block / 448 (1 where the block is all zero, NaN where it holds
    nothing but NaN poison); byte = torch's round-to-nearest float8_e4m3fn cast of x / scale.  NaN
    poison stays NaN (0x7f)."""
    P, ps, hkv, d = pages.shape
    out = torch.empty((P, ps, hkv, d), dtype=torch.uint8, device=pages.device)
    scale = torch.empty((P, hkv), dtype=torch.float32, device=pages.device)
    for i in range(0, P, chunk_pages):
        x = pages[i:i + chunk_pages].float()
        isnan = torch.isnan(x)
        amax = torch.where(isnan, torch.zeros_like(x), x.abs()).amax(dim=(1, 3))
        sc = torch.where(amax > 0, amax / E4M3_MAX, torch.ones_like(amax))
        sc = torch.where(isnan.all(dim=3).all(dim=1), torch.full_like(sc, float("nan")), sc)
        y = x / torch.where(torch.isnan(sc), torch.ones_like(sc), sc).view(-1, 1, hkv, 1)
        out[i:i + chunk_pages] = y.to(torch.float8_e4m3fn).view(torch.uint8)
        scale[i:i + chunk_pages] = sc
    return out, scale


def quantize_batch_fp8(batch: "DecodeBatch") -> Fp8DecodeBatch:
    """The same seeded batch with its cache stored as E4M3 + per-(page, kv head) scales."""
    k8, ks = _quantize_pool_e4m3(batch.k_pages)
    v8, vs = _quantize_pool_e4m3(batch.v_pages)
    return Fp8DecodeBatch(q=batch.q, k_pages=k8, v_pages=v8, k_scale=ks, v_scale=vs,
                          block_table=batch.block_table, seq_lens=batch.seq_lens,
                          softmax_scale=batch.softmax_scale, name=(batch.name + "+fp8kv") if batch.name else "fp8kv",
                          seed=batch.seed)


def to_hnd(batch: Fp8DecodeBatch) -> Fp8DecodeBatch:
    """Same cache, pools re-laid out [P, Hkv, page_size, D] (pure data movement)."""
    assert batch.kv_layout == "NHD"
    return dataclasses.replace(batch, k_pages=batch.k_pages.permute(0, 2, 1, 3).contiguous(),
                               v_pages=batch.v_pages.permute(0, 2, 1, 3).contiguous(), kv_layout="HND")


def permute_pages_fp8(batch: Fp8DecodeBatch, seed: int) -> Fp8DecodeBatch:
    """permute_pages for the FP8 cache: pages and their scale rows move together."""
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    perm = torch.randperm(batch.num_pages, generator=g)          # new_id = perm[old_id]
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(batch.num_pages)
    dev = batch.k_pages.device
    invd = inv.to(dev)
    bt = batch.block_table.cpu().to(torch.int64)
    bt2 = torch.where(bt >= 0, perm[bt.clamp_min(0)], bt).to(torch.int32)
    return dataclasses.replace(batch, k_pages=batch.k_pages[invd], v_pages=batch.v_pages[invd],
                               k_scale=batch.k_scale[invd], v_scale=batch.v_scale[invd],
                               block_table=bt2.to(dev))


def f32(x: float) -> float:
    """Round a python float to fp32 (the ABI's softmax_scale is a C float)."""
    return float(np.float32(x))


def _randn_bf16(shape, gen: torch.Generator, device, scale: float = 1.0,
                chunk_elems: int = 1 << 27) -> torch.Tensor:
    """N(0,1)*scale drawn in fp32, rounded to bf16 (RNE); chunked along dim 0 to bound memory."""
    out = torch.empty(shape, dtype=torch.bfloat16, device=device)
    if out.numel() == 0:
        return out
    row = max(1, out[0].numel())
    step = max(1, chunk_elems // row)
    for i in range(0, shape[0], step):
        n = min(step, shape[0] - i)
        x = torch.randn((n,) + tuple(shape[1:]), generator=gen, device=device, dtype=torch.float32)
        if scale != 1.0:
            x.mul_(scale)
        out[i:i + n] = x.to(torch.bfloat16)
    return out


def pages_needed(seq_len: int, page_size: int) -> int:
    return (int(seq_len) + page_size - 1) // page_size


def make_batch(seq_lens: Sequence[int], num_q_heads: int, num_kv_heads: int, head_dim: int,
               page_size: int, seed: int, device="cpu", *, k_scale: float = 1.0,
               num_pages: Optional[int] = None, max_pages_per_seq: Optional[int] = None,
               spare_tokens: int = 0, poison_unused: bool = False,
               peaked_frac: float = 0.0, peaked_offset: float = 0.0,
               softmax_scale: Optional[float] = None, name: str = "") -> DecodeBatch:
    """Build one paged decode batch.

    * Physical pages are dealt to sequences from one seeded permutation of the
      pool, so the sequences interleave in memory.
    * Each sequence owns ceil((L_b + spare_tokens) / page_size) table entries
      (the spare ones are room for appended tokens, config 5).
    * ``poison_unused``: table entries past a sequence's owned pages are -1,
      pages nobody owns are filled with NaN, and the slots past L_b in the last
      page hold NaN (parity runs); otherwise they hold ordinary random data.
    * ``peaked_frac``/``peaked_offset``: config 4's "1% of keys given a +4.0
      offset along Q's direction": per (b, kv head), u = mean of the group's G
      query vectors, normalised in fp32; positions i.i.d. Bernoulli(frac);
      k <- bf16(float(k) + offset * u).  (reading R13.)
    """
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    cpu_gen = torch.Generator(device="cpu")
    cpu_gen.manual_seed(seed)

    batch = len(seq_lens)
    owned = [pages_needed(int(l) + spare_tokens, page_size) for l in seq_lens]
    total_owned = sum(owned)
    if num_pages is None:
        num_pages = total_owned
    if max_pages_per_seq is None:
        max_pages_per_seq = max(1, max(owned))
    assert num_pages >= total_owned, (num_pages, total_owned)
    assert max_pages_per_seq >= max(owned + [0])

    q = _randn_bf16((batch, num_q_heads, head_dim), gen, device)
    k_pages = _randn_bf16((num_pages, page_size, num_kv_heads, head_dim), gen, device, k_scale)
    v_pages = _randn_bf16((num_pages, page_size, num_kv_heads, head_dim), gen, device)

    perm = torch.randperm(num_pages, generator=cpu_gen).to(torch.int32)
    fill = -1 if poison_unused else 0
    block_table = torch.full((batch, max_pages_per_seq), fill, dtype=torch.int32)
    off = 0
    for b in range(batch):
        block_table[b, :owned[b]] = perm[off:off + owned[b]]
        off += owned[b]
    lens = torch.tensor([int(l) for l in seq_lens], dtype=torch.int32)

    if peaked_frac > 0.0:
        g = num_q_heads // num_kv_heads
        for b in range(batch):
            npg = pages_needed(int(seq_lens[b]), page_size)
            if npg == 0:
                continue
            ids = block_table[b, :npg].to(device=device, dtype=torch.int64)
            qbar = q[b].float().view(num_kv_heads, g, head_dim).mean(dim=1)
            u = qbar / qbar.norm(dim=-1, keepdim=True).clamp_min(1e-20)
            mask = torch.rand((npg, page_size, num_kv_heads), generator=gen, device=device) < peaked_frac
            kk = k_pages[ids].float()
            kk += mask.unsqueeze(-1).float() * (peaked_offset * u.view(1, 1, num_kv_heads, head_dim))
            k_pages[ids] = kk.to(torch.bfloat16)
            del kk, mask

    if poison_unused:
        nan = float("nan")
        unowned = perm[off:].to(device=device, dtype=torch.int64)
        if unowned.numel():
            k_pages[unowned] = nan
            v_pages[unowned] = nan
        for b in range(batch):
            l = int(seq_lens[b])
            first_free = l  # logical token index of the first unused slot
            last_owned_tok = owned[b] * page_size
            t = first_free
            while t < last_owned_tok:
                pid = int(block_table[b, t // page_size])
                s0 = t % page_size
                k_pages[pid, s0:] = nan
                v_pages[pid, s0:] = nan
                t += page_size - s0

    if softmax_scale is None:
        softmax_scale = 1.0 / math.sqrt(head_dim)
    return DecodeBatch(q=q, k_pages=k_pages, v_pages=v_pages,
                       block_table=block_table.to(device), seq_lens=lens.to(device),
                       softmax_scale=f32(softmax_scale), name=name, seed=seed)


@dataclasses.dataclass
class PrefillBatch:
    """Inputs of the paged causal prefill (reading R20): a DecodeBatch's cache plus the ragged chunk queries."""

    q: torch.Tensor            # bf16 [total_q, Hq, D]: the chunks of all sequences back to back
    q_start: torch.Tensor      # int32 [batch + 1]
    k_pages: torch.Tensor
    v_pages: torch.Tensor
    block_table: torch.Tensor
    seq_lens: torch.Tensor     # tokens in the cache, the chunk's own included
    softmax_scale: float
    name: str = ""

    batch = property(lambda self: self.seq_lens.shape[0])
    total_q = property(lambda self: self.q.shape[0])
    num_q_heads = property(lambda self: self.q.shape[1])
    num_kv_heads = property(lambda self: self.k_pages.shape[2])
    head_dim = property(lambda self: self.q.shape[2])
    page_size = property(lambda self: self.k_pages.shape[1])

    def to(self, device) -> "PrefillBatch":
        mv = lambda t: t.to(device)
        return dataclasses.replace(self, q=mv(self.q), q_start=mv(self.q_start), k_pages=mv(self.k_pages),
                                   v_pages=mv(self.v_pages), block_table=mv(self.block_table), seq_lens=mv(self.seq_lens))

    def causal_pairs(self) -> int:
        """Number of (query, key <= pos) pairs per query head: sum_b sum_i (L_b - n_b + i + 1)."""
        lens = [int(x) for x in self.seq_lens.cpu()]
        qs = [int(x) for x in self.q_start.cpu()]
        tot = 0
        for b, L in enumerate(lens):
            n = qs[b + 1] - qs[b]
            tot += n * (L - n) + n * (n + 1) // 2
        return tot

    def algorithmic_flops(self) -> int:
        """4 * D flop per (query, key <= pos) pair and query head: the causal flops, not the dense square."""
        return 4 * self.head_dim * self.num_q_heads * self.causal_pairs()


def make_prefill_batch(seq_lens: Sequence[int], q_lens: Sequence[int], num_q_heads: int, num_kv_heads: int,
                       head_dim: int, page_size: int, seed: int, device="cpu", *, k_scale: float = 1.0,
                       poison_unused: bool = False, num_pages: Optional[int] = None,
                       max_pages_per_seq: Optional[int] = None, softmax_scale: Optional[float] = None,
                       name: str = "") -> PrefillBatch:
    """A paged cache of make_batch(seq_lens, ...) plus, per sequence, the queries of its last q_lens[b] tokens
    (N(0,1) -> bf16 from the same seeded generator family).  q_lens[b] <= seq_lens[b]."""
    assert len(seq_lens) == len(q_lens) and all(0 <= int(n) <= int(l) for n, l in zip(q_lens, seq_lens))
    base = make_batch(seq_lens, num_q_heads, num_kv_heads, head_dim, page_size, seed, device, k_scale=k_scale,
                      poison_unused=poison_unused, num_pages=num_pages, max_pages_per_seq=max_pages_per_seq,
                      softmax_scale=softmax_scale)
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(seed + 7919)
    total_q = int(sum(int(n) for n in q_lens))
    q = _randn_bf16((total_q, num_q_heads, head_dim), gen, device)
    q_start = torch.tensor([0] + list(np.cumsum([int(n) for n in q_lens])), dtype=torch.int32, device=device)
    return PrefillBatch(q=q, q_start=q_start, k_pages=base.k_pages, v_pages=base.v_pages, block_table=base.block_table,
                        seq_lens=base.seq_lens, softmax_scale=base.softmax_scale, name=name)


def sink_batch(seq_len: int, num_q_heads: int, num_kv_heads: int, head_dim: int, page_size: int, seed: int,
               device="cpu", *, sink_nats: float = 13.0, v_mean: float = 0.3, v_std: float = 0.1,
               k_scale: float = 0.05) -> DecodeBatch:
    """Stress recipe for low-precision P (input preparation only): one sequence whose token 0 is an attention sink
    `sink_nats` above a flat tail (k ~ k_scale * N(0,1)), values with a NONZERO mean (v ~ N(v_mean, v_std^2), so the
    tail's mass matters to the output and an FP8 page scale amax/448 is ~2e-3).  The G heads of a group get the same
    query, so every head sees the same sink logit: k_0 = sink_nats / (scale * |q|^2) * q."""
    b = make_batch([seq_len], num_q_heads, num_kv_heads, head_dim, page_size, seed, device, k_scale=k_scale,
                   poison_unused=True)
    g = num_q_heads // num_kv_heads
    q = b.q.view(1, num_kv_heads, g, head_dim)
    q[:] = q[:, :, :1, :]
    gen = torch.Generator(device=b.q.device)
    gen.manual_seed(seed + 1)
    npg = pages_needed(seq_len, page_size)
    ids = b.block_table[0, :npg].long()
    v = torch.randn((npg, page_size, num_kv_heads, head_dim), generator=gen, device=b.q.device) * v_std + v_mean
    v = v.to(torch.bfloat16)
    tail = npg * page_size - seq_len
    if tail:
        v.view(-1, num_kv_heads, head_dim)[seq_len:] = float("nan")
    b.v_pages[ids] = v
    qf = b.q[0].float().view(num_kv_heads, g, head_dim)[:, 0, :]
    k0 = qf * (sink_nats / (b.softmax_scale * (qf * qf).sum(-1, keepdim=True)))
    b.k_pages[int(b.block_table[0, 0]), 0] = k0.to(torch.bfloat16)
    return b


# ---------------------------------------------------------------------------
# BASELINE.json configs (C1..C5), concrete per SURVEY.md §8(d)
# ---------------------------------------------------------------------------

def ragged_lens(batch: int, lo: int, hi: int, seed: int) -> list:
    """Integers uniform on [lo, hi] inclusive from numpy's default_rng(seed)."""
    return [int(x) for x in np.random.default_rng(seed).integers(lo, hi, size=batch, endpoint=True)]


def _round_up(x: int, m: int) -> int:
    return (x + m - 1) // m * m


def config1_tiny(device="cpu", poison_unused: bool = False) -> DecodeBatch:
    """C1: batch 1, 4q/1kv, D 64, 512 tokens, ps 16, perm of exactly 32 pages; seed 1001."""
    return make_batch([512], 4, 1, 64, 16, 1001, device, num_pages=32, max_pages_per_seq=32,
                      poison_unused=poison_unused, name="C1-tiny")


def config2_agent_single(device="cpu", poison_unused: bool = False, seed: int = 1002) -> DecodeBatch:
    """C2: batch 1, 64q/8kv, D 128, 32768 tokens, ps 16, 2048 of a 4096-page pool, K*0.5."""
    return make_batch([32768], 64, 8, 128, 16, seed, device, k_scale=0.5, num_pages=4096,
                      max_pages_per_seq=2048, poison_unused=poison_unused, name="C2-agent-1x32K")


def config3_agent_ragged(device="cpu", poison_unused: bool = False, spare_tokens: int = 0,
                         lo: int = 8192, hi: int = 65536, batch: int = 32,
                         max_pages_per_seq: Optional[int] = None) -> DecodeBatch:
    """C3: batch 32, 64q/8kv, D 128, L_b ~ U[8192, 65536] (rng 1003), ps 16, shared shuffled pool."""
    lens = ragged_lens(batch, lo, hi, 1003)
    owned = sum(pages_needed(l + spare_tokens, 16) for l in lens)
    pool = _round_up(owned, 4096) + 4096
    maxp = max_pages_per_seq or max(4096, pages_needed(hi + spare_tokens, 16))
    return make_batch(lens, 64, 8, 128, 16, 1003, device, num_pages=pool,
                      max_pages_per_seq=maxp, spare_tokens=spare_tokens,
                      poison_unused=poison_unused, name="C3-agent-32xU[8K,64K]")


def config4_memory_long(device="cpu", poison_unused: bool = False, batch: int = 16,
                        context: int = 131072) -> DecodeBatch:
    """C4: batch 16, 32q/8kv, D 128, 131072 tokens each, ps 32, 1% keys +4.0 along Q; seed 1004."""
    owned = batch * pages_needed(context, 32)
    return make_batch([context] * batch, 32, 8, 128, 32, 1004, device, num_pages=owned + 4096,
                      max_pages_per_seq=max(4096, pages_needed(context, 32)),
                      poison_unused=poison_unused, peaked_frac=0.01, peaked_offset=4.0,
                      name="C4-memory-16x128K")


def config5_memory_ragged(device="cpu", poison_unused: bool = False, spare_tokens: int = 64,
                          lo: int = 65536, hi: int = 131072, batch: int = 8) -> DecodeBatch:
    """C5's memory-model batch: batch 8, 32q/8kv, D 128, L_b ~ U[65536, 131072] (rng 1005), ps 16."""
    lens = ragged_lens(batch, lo, hi, 1005)
    owned = sum(pages_needed(l + spare_tokens, 16) for l in lens)
    return make_batch(lens, 32, 8, 128, 16, 1005, device, num_pages=_round_up(owned, 4096),
                      max_pages_per_seq=pages_needed(hi + spare_tokens, 16),
                      spare_tokens=spare_tokens, poison_unused=poison_unused,
                      name="C5-memory-8xU[64K,128K]")


def decode_step_rows(batch: DecodeBatch, step: int, seed_base: int):
    """Config 5, step i: one fresh q and one new (k, v) row per sequence, seeded by
    seed_base + step so the timed loop does no RNG.  Returns (q, new_k, new_v) bf16."""
    dev = batch.q.device
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed_base + step)
    q = _randn_bf16(tuple(batch.q.shape), gen, dev)
    new_k = _randn_bf16((batch.batch, batch.num_kv_heads, batch.head_dim), gen, dev)
    new_v = _randn_bf16((batch.batch, batch.num_kv_heads, batch.head_dim), gen, dev)
    return q, new_k, new_v


def permute_pages(batch: DecodeBatch, seed: int) -> DecodeBatch:
    """Same logical cache, different physical placement: move every page through a
    seeded permutation of the pool and rewrite the block table to match."""
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    perm = torch.randperm(batch.num_pages, generator=g)          # new_id = perm[old_id]
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(batch.num_pages)
    dev = batch.k_pages.device
    k2 = batch.k_pages[inv.to(dev)]
    v2 = batch.v_pages[inv.to(dev)]
    bt = batch.block_table.cpu().to(torch.int64)
    valid = bt >= 0
    bt2 = torch.where(valid, perm[bt.clamp_min(0)], bt).to(torch.int32)
    return dataclasses.replace(batch, k_pages=k2, v_pages=v2, block_table=bt2.to(dev))


# ---------------------------------------------------------------------------------------------
# two-tier cache (PAPER.md L61 / L245: CPU offloading): input preparation only
# ---------------------------------------------------------------------------------------------
@dataclasses.dataclass
class OffloadBatch:
    """A DecodeBatch whose cold pages live in a second pool in pinned host memory.  block_table entry e >= 0 is page
    e of (k_pages, v_pages) on the device, e < 0 is page -1 - e of (k_host, v_host)."""

    base: DecodeBatch          # q, device pools, remapped block table, seq_lens
    k_host: torch.Tensor       # bf16 [P_host, page_size, Hkv, D], pinned
    v_host: torch.Tensor
    host_tokens: int           # cached tokens that live in the host pool

    def host_bytes(self) -> int:
        return self.host_tokens * self.base.num_kv_heads * self.base.head_dim * 2 * 2


def offload_pages(batch: DecodeBatch, frac: float, seed: int, coldest_first: bool = True) -> OffloadBatch:
    """Move a fraction `frac` of every sequence's USED pages to a pinned host pool and rewrite the block table
    (pure data movement, like permute_pages).  coldest_first: the oldest pages of each sequence go (what an engine
    offloads); otherwise a seeded random subset.  The device copies of the moved pages are overwritten with NaN, so a
    kernel that still read them would show it."""
    assert batch.q.is_cuda and 0.0 <= frac <= 1.0
    ps = batch.page_size
    lens = batch.seq_lens.cpu().tolist()
    bt = batch.block_table.cpu().clone()
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    moved, host_tokens = [], 0
    for b, L in enumerate(lens):
        n = pages_needed(int(L), ps)
        k = int(round(frac * n))
        if k == 0:
            continue
        pick = list(range(k)) if coldest_first else sorted(torch.randperm(n, generator=g)[:k].tolist())
        for j in pick:
            moved.append(int(bt[b, j]))
            bt[b, j] = -1 - (len(moved) - 1)
            host_tokens += min(ps, int(L) - j * ps)
    n_host = max(1, len(moved))
    shape = (n_host,) + tuple(batch.k_pages.shape[1:])
    k_host = torch.zeros(shape, dtype=torch.bfloat16).pin_memory()
    v_host = torch.zeros(shape, dtype=torch.bfloat16).pin_memory()
    k_dev, v_dev = batch.k_pages.clone(), batch.v_pages.clone()
    if moved:
        ids = torch.tensor(moved, dtype=torch.int64, device=batch.k_pages.device)
        k_host[: len(moved)].copy_(batch.k_pages[ids])
        v_host[: len(moved)].copy_(batch.v_pages[ids])
        k_dev[ids] = float("nan")
        v_dev[ids] = float("nan")
    base = dataclasses.replace(batch, k_pages=k_dev, v_pages=v_dev, block_table=bt.to(batch.block_table.device))
    return OffloadBatch(base=base, k_host=k_host, v_host=v_host, host_tokens=host_tokens)


def combined_pool_cpu(ob: OffloadBatch) -> DecodeBatch:
    """The same logical cache as ONE pool on the CPU (device pool followed by the host pool, table entries e < 0
    rewritten to P_dev - 1 - e): what the oracle, which knows one pool, is given.  Data movement only."""
    b = ob.base
    P = b.num_pages
    k = torch.cat([b.k_pages.cpu(), ob.k_host], dim=0)
    v = torch.cat([b.v_pages.cpu(), ob.v_host], dim=0)
    bt = b.block_table.cpu().to(torch.int64)
    bt = torch.where(bt < 0, P - 1 - bt, bt).to(torch.int32)
    return DecodeBatch(q=b.q.cpu(), k_pages=k, v_pages=v, block_table=bt, seq_lens=b.seq_lens.cpu(),
                       softmax_scale=b.softmax_scale, name=b.name, seed=b.seed)
