/*
 * comem_decode_attn.h — C ABI of libcomem_decode.so (B200 / sm_100a only).
 *
 * The one operation: single-query ("decode step") grouped-query attention over a
 * paged bf16 KV cache addressed through a block table, computed as split-KV
 * partial softmax + log-sum-exp combine.
 *
 * Where the operation is defined (P:Lnn = /root/reference/PAPER.md line nn):
 *   P:L49  §2.2  Q in R^{l x h_q x d_h}, K, V in R^{l x h_kv x d_h}; the KV cache
 *                [K_1; ...; K_l], [V_1; ...; V_l] kept per KV head.
 *   P:L51  fn.1  KV heads are distinct from attention heads because of GQA.
 *   P:L61  §2.2  decode step t appends one (K, V) row to the cache
 *                (comem_kv_append_async) and then reads the WHOLE cache for the
 *                one new query (comem_decode_attn*); it is memory-bound.
 *   P:L25        the cache is paged (PagedAttention is named, no layout given).
 *   P:L184 eq.5  t = L*S/W: the roofline this library is measured against.
 * The softmax-attention formula itself is not written in the paper; the
 * readings this ABI fixes are listed in DESIGN.md ("Readings", R1..R13):
 *   out[b,h,:] = sum_t softmax_t(softmax_scale * q[b,h,:].k_t[kvh,:]) * v_t[kvh,:]
 *   over t in [0, seq_lens[b]), kvh = h / (num_q_heads / num_kv_heads),
 *   (k_t, v_t) = row (page block_table[b][t / page_size], slot t % page_size).
 *
 * Conventions for every entry point
 *   - "device" pointers are CUDA device memory of the CURRENT device; "host"
 *     pointers are ordinary (preferably pinned) host memory.
 *   - The caller owns every buffer.  The library never allocates device memory,
 *     never frees and never keeps a pointer after the call returns (it caches
 *     only TMA descriptors keyed by pool address and shape).
 *   - Tensor base pointers must be 16-byte aligned (k_pages / v_pages: 128-byte).
 *   - Return value: a COMEM_* status; no exceptions or aborts cross the ABI.
 *   - Device-side DATA (seq_lens, block_table contents) is not validated:
 *     seq_lens[b] > max_pages_per_seq * page_size, or a page id outside
 *     [0, num_pages) in a USED table entry, is undefined behaviour.  Table
 *     entries j >= ceil(seq_lens[b] / page_size), slots past seq_lens[b] in the
 *     last page, and pages no sequence uses are never read semantically: the
 *     result does not depend on their contents (NaN / Inf / wild ids included).
 *   - Results are deterministic: the same logical inputs give bit-identical
 *     output regardless of physical page placement, stream, or concurrent work.
 */
#ifndef COMEM_DECODE_ATTN_H
#define COMEM_DECODE_ATTN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    COMEM_OK = 0,
    COMEM_ERR_INVALID_ARG = 1, /* null required pointer, batch <= 0, Hq % Hkv != 0, bad scale, misaligned */
    COMEM_ERR_UNSUPPORTED = 2, /* head_dim not in {64,128}; page_size not in {16,32}; G = Hq/Hkv not in 1..8;
                                  batch > COMEM_MAX_BATCH; device is not sm_100 */
    COMEM_ERR_WORKSPACE = 3,   /* workspace NULL or smaller than comem_decode_attn_workspace_bytes() */
    COMEM_ERR_CUDA = 4         /* a CUDA runtime/driver call failed (no device, launch error, ...) */
};

#define COMEM_MAX_BATCH 4096

/*
 * Per-call launch options of the attention entry points (last argument of every *_async attention call; NULL = the
 * process defaults below).  They change WHERE and HOW the kernel is launched, never its result bits' validity: the
 * split-KV schedule is a function of (seq_lens, num_kv_heads, grid_ctas), so a given grid_ctas reproduces its own
 * bits exactly and any value is within the parity tolerance.
 *   grid_ctas            > 0: size of this call's persistent decode grid (its share of the SMs: the agent batch and
 *                        the memory-model batch of the k-step-off pipeline, run side by side when their
 *                        grids sum to the SM count; comem_sm_partition picks the split).  0: the default
 *                        (comem_set_grid_ctas' value if set, else one CTA per SM).  comem_prefill_attn_async: > 0 makes the prefill
 *                        kernel persistent on that many SMs (default there: one CTA per work item).
 *   programmatic_launch  1 / 0: launch with / without programmatic stream serialization (the next launch of the
 *                        stream starts its prologue on SMs the previous one has released: shortest back-to-back steps,
 *                        but a stream's NEXT kernel then parks on every free SM; use 0 with an SM partition).
 *                        -1: the default (comem_set_programmatic_launch's value, initially 1).
 *   flags                bit set of COMEM_LAUNCH_* below; 0 = none.
 *     COMEM_LAUNCH_KV_PREFIX_IMMUTABLE   a PROMISE by the caller, for decode calls launched with programmatic stream
 *                        serialization: no work of the stream that may still be running when this call's kernel starts
 *                        (the kernels enqueued just before it) writes (a) K/V rows at positions below the last 16-token
 *                        tile of any sequence as seq_lens reads at that moment, (b) the block-table entries of the pages
 *                        holding them, (c) FP8 cache: those pages' scales.  This is what a decode loop does anyway: the
 *                        cache of old tokens never changes (the step appends K^(t), V^(t) to
 *                        the cache of steps < t), comem_kv_append_async writes one row at position seq_lens[b].  The kernel
 *                        then loads its first tiles into shared memory BEFORE it waits for the preceding kernel
 *                        (instead of only hinting them into L2), re-validating its schedule after the wait.  Results are
 *                        bit-identical with and without the flag.  If the promise is broken the call may attend stale rows.
 *     COMEM_LAUNCH_SPLIT_COMBINE        run the log-sum-exp combine as a second, small kernel launched right behind the
 *                        split kernel (2 launches; its CTAs sit beside the split kernel's and start the moment the split
 *                        grid has drained) instead of inside it.  Shortest back-to-back steps for a step of few long
 *                        segments (batch * num_kv_heads <= 64: one 32K sequence); no gain for large batches.  The combine
 *                        sums a segment's partials in a different (equally fixed) order than the fused kernel, so the
 *                        result is within rounding of the default's, and bit-identical to itself from run to run.
 *     COMEM_LAUNCH_FP8_TENSOR           comem_decode_attn_fp8_async only (COMEM_ERR_INVALID_ARG elsewhere): run the split kernel that feeds the E4M3 tiles straight to the tensor cores
 *                        (tcgen05 kind::f8f6f4, q and P each split exactly into two E4M3 parts) instead of widening
 *                        every byte to fp16 in the warps; the combine always runs as the second, dependent kernel.
 *                        head_dim 128, no sliding window, batch <= 1024 (COMEM_ERR_UNSUPPORTED otherwise).  Same
 *                        schedule and reduction structure, results within rounding of the default kernel's (P carries
 *                        8 significant bits instead of 11) and bit-identical to themselves from run to run and under
 *                        page permutation.  The other flags are accepted and ignored by this kernel.
 * Two host threads may enqueue concurrently with different options; nothing here is process state.
 */
enum { COMEM_LAUNCH_KV_PREFIX_IMMUTABLE = 1, COMEM_LAUNCH_SPLIT_COMBINE = 2, COMEM_LAUNCH_Q_STABLE = 4, COMEM_LAUNCH_FP8_TENSOR = 8 };
typedef struct {
    int grid_ctas;
    int programmatic_launch;
    int flags;
} comem_launch_opts;

/*
 * comem_decode_attn_async — enqueue one decode-attention step on `cuda_stream`.
 *
 * Enqueue-only: no host synchronisation, no device->host copy, no allocation;
 * safe inside CUDA-graph capture.  Launches 1 kernel: the split-KV kernel, in which the
 * last CTA to finish a cut (b, kv head) segment also runs the log-sum-exp combine for it.
 * Returns launch-time errors only.
 *
 *   q            device, bf16 [batch][num_q_heads][head_dim], contiguous
 *   k_pages      device, bf16 [num_pages][page_size][num_kv_heads][head_dim]
 *   v_pages      device, same shape, separate allocation
 *   block_table  device, int32 [batch][max_pages_per_seq]; entry j = physical page
 *                of logical page j of that sequence
 *   seq_lens     device, int32 [batch]; tokens valid in each sequence (0 allowed:
 *                that row of out is +0.0 and its lse is -inf)
 *   softmax_scale  fp32, finite, >= 0; applied to the fp32 dot product
 *   out          device, bf16 [batch][num_q_heads][head_dim]; fp32 accumulate,
 *                round-to-nearest-even
 *   lse_out      device, fp32 [batch][num_q_heads] natural-log log-sum-exp of the
 *                scaled logits, or NULL
 *   workspace    device scratch of >= comem_decode_attn_workspace_bytes(...) bytes,
 *                256-byte aligned.  Holds the per-segment arrival counters and the
 *                split partials.  The counters must be zero when a call starts:
 *                run comem_workspace_init_async once on a fresh (or foreign-written)
 *                buffer; every call that completes leaves them zero again, so the
 *                same workspace serves any number of later calls of any shape it is
 *                large enough for.  Calls that may run concurrently (different
 *                streams) need DIFFERENT workspaces.
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream)
 */
int comem_decode_attn_async(const void *q, const void *k_pages, const void *v_pages,
                            const int32_t *block_table, const int32_t *seq_lens,
                            int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                            float softmax_scale, void *out, int batch, int max_pages_per_seq,
                            int64_t num_pages, float *lse_out, void *workspace,
                            size_t workspace_bytes, void *cuda_stream, const comem_launch_opts *opts);

/*
 * comem_workspace_init_async — zero the arrival counters at the head of `workspace`
 * (one cudaMemsetAsync of workspace_bytes' counter prefix on `cuda_stream`).  Needed once
 * per buffer, before its first use (see `workspace` above).  The prefix length depends only
 * on (batch, num_kv_heads); pass the largest shape the buffer will serve.
 */
int comem_workspace_init_async(void *workspace, size_t workspace_bytes, int batch, int num_q_heads,
                               int num_kv_heads, int head_dim, void *cuda_stream);

/*
 * comem_decode_attn_phases_async — the same step with its two phases as separate kernels:
 * COMEM_PHASE_SPLIT alone runs K1 un-fused (page-gather + QK^T + online softmax + PV; writes
 * finished rows and the split partials into `workspace`, merges nothing), COMEM_PHASE_COMBINE
 * alone runs K2 (stand-alone LSE merge of the partials in `workspace`; also writes the rows of
 * empty sequences).  SPLIT|COMBINE is comem_decode_attn_async (one fused launch).  The
 * two-call form (same arguments, same workspace, same stream order) gives a result within
 * rounding of the fused one (K2 sums the partials in 4 interleaved stripes, the fused merge in
 * plain split order); tests use it to check K2 and the partial format on their own.
 */
enum { COMEM_PHASE_SPLIT = 1, COMEM_PHASE_COMBINE = 2 };
int comem_decode_attn_phases_async(const void *q, const void *k_pages, const void *v_pages,
                                   const int32_t *block_table, const int32_t *seq_lens,
                                   int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                                   float softmax_scale, void *out, int batch,
                                   int max_pages_per_seq, int64_t num_pages, float *lse_out,
                                   void *workspace, size_t workspace_bytes, void *cuda_stream,
                                   int phases, const comem_launch_opts *opts);

/*
 * comem_decode_attn_window_async — the byte-reducing variant the paper calls orthogonal (sliding
 * window + attention sinks; reading R17): the query, which sits at
 * position seq_lens[b] - 1, attends only the positions t < sink_tokens and t >= seq_lens[b] - window,
 * and only the 16-token tiles holding such a position are scheduled and read.  window <= 0 (or
 * >= seq_lens[b]) means no window: the call is then comem_decode_attn_async.  sink_tokens >= 0.
 * Everything else (arguments, workspace, determinism, one fused launch) as comem_decode_attn_async;
 * the contents of positions outside the kept set never matter (NaN / Inf included).
 */
int comem_decode_attn_window_async(const void *q, const void *k_pages, const void *v_pages,
                                   const int32_t *block_table, const int32_t *seq_lens,
                                   int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                                   float softmax_scale, void *out, int batch,
                                   int max_pages_per_seq, int64_t num_pages, float *lse_out,
                                   void *workspace, size_t workspace_bytes, void *cuda_stream,
                                   int window, int sink_tokens, const comem_launch_opts *opts);

/*
 * comem_decode_attn_fp8_async — the same step over an FP8 KV cache, the other byte-reducing variant
 * the paper calls orthogonal ("KV Cache Quantization"; reading R18): half the bytes
 * per token on the same HBM roofline.
 *   k_pages, v_pages  OCP FP8 E4M3 bytes [num_pages, page_size, num_kv_heads, head_dim], device,
 *                     128-byte aligned (bias 7, max 448, 0x7f / 0xff = NaN, no infinities)
 *   k_scale, v_scale  fp32 [num_pages, num_kv_heads], device: token row (pid, slot, kvh) of K is
 *                     k_scale[pid][kvh] * e4m3(k_pages[pid][slot][kvh][:]); V likewise.  Only the scales
 *                     of pages holding a kept token are read; they must be finite.
 *   window, sink_tokens   as comem_decode_attn_window_async (window <= 0: full attention)
 *   kv_layout         COMEM_KV_LAYOUT_NHD: pools are [num_pages, page_size, num_kv_heads, head_dim] as above;
 *                     COMEM_KV_LAYOUT_HND: [num_pages, num_kv_heads, page_size, head_dim] -- a (page, kv head)
 *                     tile is then 16 x 128 B CONTIGUOUS in DRAM instead of 16 rows at a num_kv_heads*128 B pitch,
 *                     which this part's HBM serves measurably faster (FP8 variant)
 * q, out, lse_out, block_table, seq_lens, workspace, stream, determinism and the error contract are
 * those of comem_decode_attn_async.  Arithmetic: E4M3 widens exactly to fp16 and the tensor op runs in
 * fp16 with fp32 accumulation; q is converted bf16 -> fp16 (exact for 2^-14 <= |q| < 65504) and
 * p * v_scale is rounded to fp16.  head_dim 64 or 128.
 */
enum { COMEM_KV_LAYOUT_NHD = 0, COMEM_KV_LAYOUT_HND = 1 };
int comem_decode_attn_fp8_async(const void *q, const void *k_pages, const void *v_pages,
                                const float *k_scale, const float *v_scale,
                                const int32_t *block_table, const int32_t *seq_lens,
                                int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                                float softmax_scale, void *out, int batch, int max_pages_per_seq,
                                int64_t num_pages, float *lse_out, void *workspace,
                                size_t workspace_bytes, void *cuda_stream, int window, int sink_tokens,
                                int kv_layout, const comem_launch_opts *opts);

/*
 * comem_decode_attn_offload_async — the decode step over a TWO-TIER cache: part of the pages live in HBM, the cold part
 * in pinned host memory ("part of the KV cache will be either emitted or offloaded to CPU ... CPU offload is often a
 * better strategy"; every latency result of the paper is reported with and without CPU offloading, P:L245,
 * Table 1).  Nothing is copied back first: the page-gather loader issues the same TMA tile load against a
 * second tensor map over the host pool, so a host-resident page crosses the host link exactly once, straight into
 * shared memory, interleaved with the HBM-resident pages of the same sequence.
 *   k_pages_host, v_pages_host   bf16 [num_pages_host][page_size][num_kv_heads][head_dim], HOST pointers to pinned,
 *                    device-mapped memory (cudaHostAlloc / cudaHostRegister; torch's pin_memory()), 128-byte aligned
 *   block_table      entry e >= 0: physical page e of the device pool (k_pages / v_pages);
 *                    entry e <  0: physical page -1 - e of the host pool
 * Everything else -- q, out, lse_out, seq_lens, workspace, stream, launch options, determinism (bit-identical results
 * wherever a page lives: placement never enters the arithmetic) and the error contract -- as comem_decode_attn_async.
 * bf16 cache, full attention (no window) in this version.  COMEM_ERR_INVALID_ARG if a host pool is not pinned + mapped.
 */
int comem_decode_attn_offload_async(const void *q, const void *k_pages, const void *v_pages,
                                    const void *k_pages_host, const void *v_pages_host,
                                    const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                                    int num_kv_heads, int head_dim, int page_size, float softmax_scale, void *out,
                                    int batch, int max_pages_per_seq, int64_t num_pages, int64_t num_pages_host,
                                    float *lse_out, void *workspace, size_t workspace_bytes, void *cuda_stream,
                                    const comem_launch_opts *opts);

/*
 * comem_pages_copy_async — move whole pages between two pools of the same page shape (HBM <-> pinned host memory:
 * offloading cold pages, bringing them back; or compaction inside one tier).  For i in [0, n_pages): page src_ids[i] of
 * (k_src, v_src) is copied to page dst_ids[i] of (k_dst, v_dst); src_ids / dst_ids are device int32 arrays; pools may
 * be device pointers or pinned, device-mapped host pointers; page_bytes = page_size * num_kv_heads * head_dim * element
 * size, a multiple of 16.  One kernel on `cuda_stream` (it reads and writes host memory itself: no copy engine, no
 * per-page cudaMemcpy); the caller updates the block table.  Destination pages must be distinct.
 */
int comem_pages_copy_async(const void *k_src, const void *v_src, void *k_dst, void *v_dst, const int32_t *src_ids,
                           const int32_t *dst_ids, int n_pages, size_t page_bytes, void *cuda_stream);

/*
 * comem_kv_append_fp8_async — comem_kv_append_async for the FP8 cache of comem_decode_attn_fp8_async (P:L61 for
 * reading R18's cache): the new token's bf16 K row of kv head h is stored as
 *     byte = e4m3( (float)new_k[b][h][d] / k_scale[pid][h] )      pid = block_table[b][seq_lens[b] / page_size]
 * — the IEEE fp32 quotient rounded to nearest even, saturating at +-448 — V likewise with v_scale, then
 * seq_lens[b] += 1.  The page's scales are read, never written: choosing them (calibration, first-row amax, …)
 * is the caller's policy, and a page must have its scales set before its first row is appended.
 * new_k / new_v: bf16 [batch, num_kv_heads, head_dim], device.  kv_layout as above.  Enqueue-only.
 */
int comem_kv_append_fp8_async(void *k_pages, void *v_pages, const float *k_scale, const float *v_scale,
                              const int32_t *block_table, int32_t *seq_lens, const void *new_k,
                              const void *new_v, int num_kv_heads, int head_dim, int page_size, int batch,
                              int max_pages_per_seq, int kv_layout, void *cuda_stream);

/*
 * k-step-off pipeline schedule and latency model — HOST functions, no device work.
 *
 * comem_kstep_plan — Algorithm 1 for agent steps t = 1 .. num_steps with retain-turns k:
 * events[t-1] says whether a finished memory job is adopted at the start of step t (lines 4-7: s <- result,
 * KV cache invalidated), which summary is then in use (summary_upto = u: s = f(tau_{<= u}), 0 = none yet;
 * the raw buffer is tau_{u+1 : t}, eq. 4), whether the prefill is full-context (lines 9-13; also true
 * at step 1, when nothing is cached) and whether a memory job is launched after the step (lines 19-21,
 * t mod k = 0, input tau_{<= t}).  mem_delay = agent steps until a launched job counts as complete; <= 0
 * means k ("available at the start of the next cycle"); > k is COMEM_ERR_INVALID_ARG (line 20 would
 * overwrite a job in flight, which the paper leaves undefined; reading R19).
 * `events` is caller-owned, num_steps entries.
 *
 * comem_kstep_context_lengths — token counts per step for turns of turn_tokens tokens and summaries of
 * summary_tokens tokens: the agent's context under CoMem (summary + raw buffer), under the full-context
 * baseline (tau_{<= t}) and the memory model's input where a job is launched (else 0).
 *
 * comem_decode_saving_seconds (eq. 5), comem_net_speedup (eq. 6, returns 0 / 1),
 * comem_max_compression_ratio (eq. 7): S in GB per token, W in GB/s, P in tokens/s, Y in tokens.
 */
typedef struct {
    int32_t step;              /* t, 1-based */
    int32_t summary_upto;      /* u */
    uint8_t adopt_summary;
    uint8_t prefill_uncached;
    uint8_t launch_memory;
    uint8_t reserved;
} comem_kstep_event;
int comem_kstep_plan(int num_steps, int k, int mem_delay, comem_kstep_event *events);
int comem_kstep_context_lengths(const comem_kstep_event *events, int num_steps, int turn_tokens,
                                int summary_tokens, int32_t *comem_ctx, int32_t *full_ctx,
                                int32_t *memory_input);
double comem_decode_saving_seconds(double l_full, double l_sum, double s_gb_per_token, double w_gb_per_s);
int comem_net_speedup(double y_tokens, double l_full, double l_sum, double s_gb_per_token,
                      double w_gb_per_s, double p_tokens_per_s);
double comem_max_compression_ratio(double w_gb_per_s, double y_tokens, double s_gb_per_token,
                                   double p_tokens_per_s);

/*
 * comem_kstep_step_async — ONE agent step of Algorithm 1 as the library's host scheduler: everything
 * the attention path does for step t is enqueued, on two streams, from the plan entry of comem_kstep_plan:
 *   agent stream   lines 4-7   adopt a finished summary: the KV cache is invalid, the context becomes
 *                              summary + raw buffer (eq. 4): seq_lens[b] <- ctx_t for every sequence
 *                  lines 9-13  prefill attention (comem_prefill_attn_async) of the NEW tokens: the whole context
 *                              when the plan says uncached ("a full uncached prefill is required"), else
 *                              the last turn_tokens only (cached, incremental)
 *                  line 15     decode_tokens times: comem_kv_append_async + comem_decode_attn_async
 *   memory stream  lines 19-21 if the plan launches a memory job after this step: wait for the agent's step, then
 *                              the memory model's uncached prefill over tau_{<=t} (t * turn_tokens tokens) and
 *                              memory_decode_tokens decode steps (the summary it writes), behind an event
 * Sharing the GPU: while a memory job is in flight (the scheduler asks the job's completion event, without blocking)
 * both models' decode grids are sized by comem_sm_partition from the bytes each streams per step and launched without
 * programmatic serialization, so an agent step never queues behind a whole memory step; otherwise the agent has
 * every SM and programmatic launch.  This is the attention path of one layer: projections, MLPs and sampling are
 * the serving engine's; K/V rows of prefilled tokens are whatever the pools hold (the engine writes them).
 *
 * comem_kstep_model describes one model's buffers (all device pointers, caller-owned, contiguous):
 *   q_decode / out_decode   bf16 [batch][Hq][D];  new_k / new_v  bf16 [batch][Hkv][D] (the row each decode token appends)
 *   q_prefill / out_prefill bf16 [prefill_cap][Hq][D], prefill_cap >= batch * (largest context this model prefills)
 *   k_pages, v_pages, block_table, seq_lens, workspace: as comem_decode_attn_async;  q_start int32 [batch + 1]
 * The call writes seq_lens and q_start (a small kernel), out_decode, out_prefill and the workspace; it never
 * synchronizes.  stats (optional, host) reports what was enqueued.  COMEM_ERR_INVALID_ARG: a context that does not
 * fit max_pages_per_seq * page_size or prefill_cap, null buffers, decode_tokens < 0.
 */
typedef struct {
    void *q_decode, *out_decode, *q_prefill, *out_prefill, *new_k, *new_v;
    void *k_pages, *v_pages;
    int32_t *block_table, *seq_lens, *q_start;
    void *workspace;
    size_t workspace_bytes;
    int64_t num_pages, prefill_cap;
    int batch, num_q_heads, num_kv_heads, head_dim, page_size, max_pages_per_seq;
    float softmax_scale;
} comem_kstep_model;
typedef struct {
    int32_t agent_ctx;            /* tokens in the agent's context at this step (eq. 4) */
    int32_t agent_prefill_tokens; /* per sequence: ctx if uncached, else turn_tokens */
    int32_t memory_ctx;           /* tokens the memory job prefills (0 if none launched) */
    int32_t agent_grid, memory_grid; /* decode grids used (0 = default: every SM) */
    int32_t memory_in_flight;     /* 1 if the SM partition was applied to the agent's decode steps */
    int32_t launches;             /* kernels enqueued by this call */
} comem_kstep_step_stats;
int comem_kstep_step_async(const comem_kstep_event *event, int turn_tokens, int summary_tokens, int decode_tokens,
                           int memory_decode_tokens, const comem_kstep_model *agent,
                           const comem_kstep_model *memory /* NULL: no memory model on this GPU */,
                           void *agent_stream, void *memory_stream, void *memory_done_event /* cudaEvent_t */,
                           void *agent_step_event /* cudaEvent_t */, comem_kstep_step_stats *stats);

/*
 * comem_prefill_attn_async — causal prefill attention over the paged cache: the compute-bound
 * step of the path.  P:L149-156 (Algorithm 1 lines 9-13): "Prefill new tokens only" when the KV cache is valid
 * (cached, incremental prefill), "Prefill full context" after a summary adoption invalidated it (uncached);
 * P:L57-59 (§2.2: prefill is compute-bound, it sets TTFT); P:L122 (§3.2: "a full uncached prefill is required"
 * after every adoption); P:L245 (chunked prefill + prefix caching in the paper's serving engine).  The formula is
 * DESIGN.md reading R20: sequence b holds seq_lens[b] = L_b cached tokens, the LAST n_b = q_start[b+1] - q_start[b]
 * of which are the new ones (their K/V rows are already in the cache); query i of the chunk sits at position
 * pos = L_b - n_b + i and attends the keys t <= pos:
 *     out[q_start[b] + i, h, :] = sum_{t <= pos} softmax_t(softmax_scale * q[q_start[b] + i, h, :] . k_t[kvh, :]) v_t[kvh, :]
 * n_b = 1 is the decode step; n_b = L_b is the uncached full prefill; n_b = 0 contributes no rows.
 *
 *   q            device, bf16 [total_q][num_q_heads][head_dim], contiguous: the chunks of all sequences back to back
 *   q_start      device, int32 [batch + 1], q_start[0] = 0, non-decreasing, q_start[batch] = total_q;
 *                n_b <= seq_lens[b] (a longer chunk is undefined behaviour, like every other device-side datum)
 *   out          device, bf16 [total_q][num_q_heads][head_dim]; lse_out device fp32 [total_q][num_q_heads] or NULL
 *   total_q      host copy of q_start[batch] (sizes the grid and the q tensor map)
 *   k_pages, v_pages, block_table, seq_lens, softmax_scale, num_pages, max_pages_per_seq: as comem_decode_attn_async
 * Shapes: head_dim 64 or 128, page_size 16 or 32, G = num_q_heads / num_kv_heads <= 16.
 * Enqueue-only, 1 kernel (tcgen05 tensor cores, accumulators in tensor memory), no workspace.  Deterministic: a row
 * is reduced by one thread in logical token order; physical page placement never enters the arithmetic.
 * Arithmetic: bf16 x bf16 -> fp32 on the tensor cores, softmax in fp32 (log2 domain), P rounded to bf16 for the
 * second product with the normaliser summed from the ROUNDED p (reading R16), bf16 output, round-to-nearest-even.
 */
int comem_prefill_attn_async(const void *q, const void *k_pages, const void *v_pages,
                             const int32_t *block_table, const int32_t *seq_lens, const int32_t *q_start,
                             int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                             float softmax_scale, void *out, int batch, int total_q, int max_pages_per_seq,
                             int64_t num_pages, float *lse_out, void *cuda_stream, const comem_launch_opts *opts);

/*
 * comem_decode_attn_static_async — comem_decode_attn_async for callers that cannot allocate device memory (code under
 * CUDA-graph capture, serving loops and harnesses that forbid cudaMalloc): the same decode-attention step (
 * the same kernels, the same schedule, results bit-identical to comem_decode_attn_async with the same options), with
 * its scratch (arrival counters + split partials) in a device array that is part of the library image instead of a
 * caller-provided workspace.  It calls no cudaMalloc / cudaFree and no allocating library routine; the caller passes
 * only inputs and outputs.  Arguments as comem_decode_attn_async, without `workspace`.
 *
 * Limits and sharing:
 *   - the array is COMEM_STATIC_SCRATCH_BYTES (12 MiB) of device memory on EVERY GPU the process loads the library on,
 *     held until the process exits; comem_static_scratch_bytes() returns the figure;
 *   - a shape is accepted iff comem_decode_attn_workspace_bytes(batch, num_q_heads, num_kv_heads, head_dim, ..) <=
 *     COMEM_STATIC_SCRATCH_BYTES (e.g. batch <= 64 at 64 q heads / 8 kv heads / head_dim 128; batch <= 256 at 16 / 4);
 *     a larger shape returns COMEM_ERR_WORKSPACE and enqueues nothing;
 *   - every call on a device shares the one array, which keeps the previous call's contents: each call first enqueues a
 *     cudaMemsetAsync of the counter prefix (<= 64 KiB) on `cuda_stream`, then the kernel(s).  Calls that may OVERLAP on
 *     the GPU (different streams, or graphs replayed concurrently) RACE on it: serialise them, or give the others a
 *     workspace of their own through comem_decode_attn_async;
 *   - the array's device address is looked up on the first call on each device (cudaGetSymbolAddress, with that device
 *     current): make that first call outside stream capture.
 */
#define COMEM_STATIC_SCRATCH_BYTES (12 * 1024 * 1024)
size_t comem_static_scratch_bytes(void);
int comem_decode_attn_static_async(const void *q, const void *k_pages, const void *v_pages,
                                   const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                                   int num_kv_heads, int head_dim, int page_size, float softmax_scale, void *out,
                                   int batch, int max_pages_per_seq, int64_t num_pages, float *lse_out,
                                   void *cuda_stream, const comem_launch_opts *opts);

/* Same on the legacy default stream, then cudaStreamSynchronize: also returns
 * execution errors (COMEM_ERR_CUDA). */
int comem_decode_attn(const void *q, const void *k_pages, const void *v_pages,
                      const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                      int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                      void *out, int batch, int max_pages_per_seq, int64_t num_pages,
                      float *lse_out, void *workspace, size_t workspace_bytes);

/* Scratch bytes needed by the calls above and below for this problem shape.
 * Pure host arithmetic (no CUDA call); depends only on the arguments. */
size_t comem_decode_attn_workspace_bytes(int batch, int num_q_heads, int num_kv_heads,
                                         int head_dim, int page_size, int max_pages_per_seq);

/*
 * comem_kv_append_async — the step before attention (P:L61,
 * K_cache^(t) = [K_cache^(t-1); K^(t)]): for every sequence b write new_k[b], new_v[b]
 * (device, bf16 [batch][num_kv_heads][head_dim]) at logical position seq_lens[b]
 * (page block_table[b][seq_lens[b] / page_size], which the caller must already have
 * placed in the table), then seq_lens[b] += 1 on the device.  Enqueue-only, 1 kernel.
 */
int comem_kv_append_async(void *k_pages, void *v_pages, const int32_t *block_table,
                          int32_t *seq_lens, const void *new_k, const void *new_v,
                          int num_kv_heads, int head_dim, int page_size, int batch,
                          int max_pages_per_seq, void *cuda_stream);

/*
 * comem_decode_step_host — one whole decode step driven from HOST buffers: the
 * end-to-end call bench.py's "e2e" times.  The KV cache is the model's resident
 * state and stays in HBM (decode waits "for the KV cache to arrive from
 * HBM"); what a step brings from the host is the new token's q, k, v rows and
 * what it returns is the attention output.
 *
 *   q_host                  host, bf16 [batch][num_q_heads][head_dim]
 *   new_k_host, new_v_host  host, bf16 [batch][num_kv_heads][head_dim], or both
 *                           NULL to skip the append
 *   out_host                host, bf16 [batch][num_q_heads][head_dim]
 *   lse_host                host, fp32 [batch][num_q_heads], or NULL
 *   k_pages, v_pages, block_table, seq_lens, workspace: device, as above
 *
 * Two paths, chosen per call with cudaPointerGetAttributes:
 *   - every host buffer is PINNED and device-mapped (cudaHostAlloc / cudaHostRegister): the kernels
 *     move the bytes themselves -- K3 reads q / new_k / new_v over the host link (q is staged in
 *     the workspace), the attention kernel stores out (and lse) straight into host memory;
 *     2 launches + cudaStreamSynchronize, no copy engine;
 *   - otherwise (pageable memory): cudaMemcpyAsync H2D(q, new_k, new_v) -> kv_append -> decode_attn
 *     -> cudaMemcpyAsync D2H(out[, lse]) -> cudaStreamSynchronize.
 * Both are host-synchronous and return execution errors too.
 */
int comem_decode_step_host(const void *q_host, const void *new_k_host, const void *new_v_host,
                           void *k_pages, void *v_pages, const int32_t *block_table,
                           int32_t *seq_lens, int num_q_heads, int num_kv_heads, int head_dim,
                           int page_size, float softmax_scale, void *out_host, int batch,
                           int max_pages_per_seq, int64_t num_pages, float *lse_host,
                           void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * comem_decode_step_host_fp8 — comem_decode_step_host for the FP8 cache (reading R18): the new token's bf16 q, k, v rows
 * come from host buffers, k / v are quantised into the E4M3 pools with the page's scales (comem_kv_append_fp8_async's
 * arithmetic), seq_lens += 1, comem_decode_attn_fp8_async runs, out (and lse) go back to the host.  Same two paths
 * (pinned + mapped: the kernels move the bytes, 2 launches + synchronize; pageable: cudaMemcpyAsync staging), same
 * host-synchronous contract.  new_k_host / new_v_host are required (this call always appends).
 */
int comem_decode_step_host_fp8(const void *q_host, const void *new_k_host, const void *new_v_host, void *k_pages,
                               void *v_pages, const float *k_scale, const float *v_scale,
                               const int32_t *block_table, int32_t *seq_lens, int num_q_heads, int num_kv_heads,
                               int head_dim, int page_size, float softmax_scale, void *out_host, int batch,
                               int max_pages_per_seq, int64_t num_pages, float *lse_host, void *workspace,
                               size_t workspace_bytes, void *cuda_stream, int kv_layout);

/*
 * Split-KV schedule introspection (host arithmetic mirroring the device
 * scheduler; used by tests and DESIGN.md).  Given host copies of seq_lens,
 * writes for each CTA i in [0, *num_ctas) its half-open range of 16-token tiles
 * [tile_begin[i], tile_begin[i+1]) in the linearised (b, kv_head, tile) order.
 * tile_begin must hold grid_ctas + 1 entries.  Returns COMEM_OK.  (Full attention only: no window.)
 */
int comem_schedule_host(const int32_t *seq_lens_host, int batch, int num_kv_heads, int grid_ctas,
                        int64_t *tile_begin, int *num_ctas);

/*
 * comem_validate_inputs — debug aid for the one thing the hot path trusts (see "Device-side DATA"
 * above): checks on the device that 0 <= seq_lens[b] <= max_pages_per_seq * page_size and that every
 * USED block-table entry is a page id in [0, num_pages).  Host-synchronous (1 kernel, a 4-byte
 * read-back through `workspace`, which may be the attention workspace).  Returns COMEM_OK or
 * COMEM_ERR_INVALID_ARG.  With the environment variable COMEM_DEBUG_VALIDATE=1 the synchronous
 * entry points (comem_decode_attn, comem_decode_step_host) run it first and return its verdict
 * instead of computing on bad data; the *_async entry points never validate.
 * COMEM_DEBUG_STALE_GUESS=1 (read once per process) is a testing aid for the decode kernel's recovery paths: every launch
 * computes its first, speculative split-KV schedule from lengths 16 tokens short -- as if the append kernel queued before
 * it had not run yet -- so the validation after the wait fails on every launch and the schedule is recomputed (classic
 * order) or the early attempt aborted and rerun (COMEM_LAUNCH_KV_PREFIX_IMMUTABLE).  Results are unchanged, bit for bit.
 */
int comem_validate_inputs(const int32_t *block_table, const int32_t *seq_lens, int batch,
                          int max_pages_per_seq, int page_size, int64_t num_pages, void *workspace,
                          size_t workspace_bytes, void *cuda_stream);

/* Persistent-grid size (CTAs) the split kernel uses on the current device, or a negative COMEM_ERR_* value. */
int comem_grid_ctas(int head_dim);

/*
 * comem_sm_partition — launch policy for two batches that share one GPU (the agent's decode step and the memory
 * model's, P:L130-176 / P:L245): split num_sms CTAs in proportion to the bytes each batch has to
 * stream, so that both persistent grids are resident together and finish together (the path is HBM-bound and an SM
 * pulls a fixed rate); each side gets at least min_ctas.  Pass the results as comem_launch_opts.grid_ctas with
 * programmatic_launch = 0.  Host arithmetic only.  *ctas_a + *ctas_b == num_sms.
 */
int comem_sm_partition(double bytes_a, double bytes_b, int num_sms, int min_ctas, int *ctas_a, int *ctas_b);

/*
 * DEPRECATED process-wide defaults, read at enqueue time by calls whose comem_launch_opts is NULL (or leaves the
 * field at its "default" value).  Two threads that need different settings must pass comem_launch_opts instead.
 * comem_set_grid_ctas(n > 0) overrides the default grid (n <= 0 restores one CTA per SM);
 * comem_set_programmatic_launch(0 / 1) switches programmatic stream serialization off / on (default 1).
 */
int comem_set_grid_ctas(int n);
int comem_set_programmatic_launch(int enabled);

/*
 * comem_read_ceiling_async — measurement aid: a hand-written read-only sum-reduction over `bytes`
 * bytes of device memory at `buf` (128-byte aligned, >= 8 KiB; use >= 8 GiB so that nothing is served from L2), the
 * ceiling eq. 5's W can reach on this part for a kernel that reads every byte once.  variant 0: 16-byte
 * vector loads, 2 x 1024 threads per SM; variant 1: the attention kernel's own transport (one CTA per SM, TMA bulk
 * copies into a 16-stage shared-memory ring, 128 KiB in flight per SM).  `sink`: device, COMEM_READ_CEILING_SINK_WORDS
 * 64-bit words that receive per-CTA sums (so no load can be elided).  Enqueue-only; time it with events on the stream.
 */
#define COMEM_READ_CEILING_SINK_WORDS 1024
int comem_read_ceiling_async(const void *buf, size_t bytes, unsigned long long *sink, int variant, void *cuda_stream);

const char *comem_status_string(int status);
int comem_version(void);

#ifdef __cplusplus
}
#endif
#endif /* COMEM_DECODE_ATTN_H */
