// decode_split.cu — K1, the whole decode-attention step in one launch: split-KV scheduler,
// page-gather loader, QK^T, online softmax, PV, partial write and (fused) the log-sum-exp combine
// for one decode step of paged GQA attention.
//
// Shape of the kernel (sm_100a):
//   * persistent grid, ONE CTA per SM (12 warps launched at 144 registers -- the producer warpgroup then hands registers
//     to the two consumer warpgroups, setmaxnreg 72 / 176 -- and ~214 KiB of shared memory), one contiguous range
//     of 16-token tiles per CTA (schedule.cuh);
//   * before griddepcontrol.wait (i.e. under the previous kernel's tail): mbarrier init, tensor-map
//     prefetch, an L2 prefetch of the small control inputs (seq_lens, block table, q), the whole
//     schedule computed SPECULATIVELY from seq_lens as it reads now (validated after the wait),
//     and a TMA L2 prefetch of the CTA's first 16 tiles;
//   * warps 8..11 = producers: each reads the block table 32 entries at a time and issues, for
//     every fourth tile of the CTA, one TMA tiled load for K and one for V ([16 tokens][D] of one kv
//     head, 128-byte swizzle) into a 16-stage shared-memory ring guarded by full/empty
//     mbarriers -- 128 KiB of K+V in flight per SM (one producer lane is issue-rate bound);
//   * warps 0..7 = consumers: tile n of the CTA goes to warp n % 8, so eight independent
//     online-softmax states stream concurrently.  Per tile and warp:
//        S[G(pad 16) x 16 tok] = Q_g K^T      mma.sync m16n8k16 (Q fragments live in registers)
//        m, p = online softmax in the log2 domain (quad shuffles for the row max)
//        O^T[D x G] += V^T P^T                mma.sync with V^T via ldmatrix.trans; P is
//                                             rounded to bf16 and l sums the ROUNDED p, so
//                                             out is an exact weighted mean of V rows;
//   * S6, at the end of a (b, kv head) segment: the eight warp states are merged through shared
//     memory in warp-index order (warp w -> query head w, lane -> one float4 of the row) and
//     either written as the final bf16 row (the CTA owned the whole segment) or as an fp32
//     partial record (acc[8][D], then one 32-byte state sector {m, l, lx} per head);
//   * S7, fused: the CTA then fences, takes a ticket on the segment's arrival counter, and the
//     CTA that arrives LAST pulls all of the segment's records with TMA bulk copies and merges
//     them in CTA-index order (merge.cuh), re-arming the counter for the next launch.  No CTA
//     ever waits for another one.  With fuse_combine == 0 the kernel stops after S6 and the
//     stand-alone K2 (combine.cu) does the merge.
//   * EARLY MODE (launch flags COMEM_LAUNCH_KV_PREFIX_IMMUTABLE [| COMEM_LAUNCH_Q_STABLE]): the
//     CTA does not sit in griddepcontrol.wait while the previous kernel drains -- its producers stream, and its
//     consumers fold, every tile below the sequence's last one from the guessed schedule; the wait, the validation
//     of the guess and a verdict on an mbarrier come at the first tile (or store) that needs the previous kernel's
//     results; a wrong guess aborts the attempt and reruns it in the classic order.  Same bits either way.
//     The mode lives in its own instance of the kernel (template parameter kEarly), launched only when the flag is set.
// The path is HBM-bound (G flop per byte); the legacy-shape tensor op is used only because at
// G = 8 the plain-FMA roofline sits below the HBM roofline ("Why mma.sync").
#ifndef COMEM_BF16_PRODUCER_WARPS
#define COMEM_BF16_PRODUCER_WARPS 4  // measured on config 2: 2 -> 25.8 us, 4 -> 25.4 us per step (faster ring fill after the PDL wait)
#endif
#ifndef COMEM_FP8_TILES_PER_PASS
#define COMEM_FP8_TILES_PER_PASS 1
#endif
#ifndef COMEM_PREFETCH_TILES
#define COMEM_PREFETCH_TILES 16
#endif
#include "decode_params.cuh"
#include "ptx.cuh"
#include "schedule.cuh"
#include "merge.cuh"
#include <type_traits>

namespace comem {

namespace {

constexpr int kConsumerWarps = 8;
constexpr int kK1LaunchRegs = 144;  // see Cfg::kLaunchRegs
constexpr int kConsumerThreads = kConsumerWarps * 32;
static_assert(kConsumerWarps == kMaxGroup, "S6 and merge.cuh map warp w to query head w of the group");
constexpr int kPrefetchTiles = COMEM_PREFETCH_TILES;  // per CTA, L2-prefetched before the PDL wait (<= 32: one per lane)
constexpr unsigned kFull = 0xffffffffu;
constexpr int kFp8PShift = 14;  // FP8 cache: p * f * 2^(ev - eref) * 2^14 < 2 * 2^14 stays below fp16's 65504 (S4)

// kFp8: the FP8 (E4M3 + per-page, per-kv-head scale) cache of reading R18.  Tiles are half the bytes,
// so the ring has twice the stages (same 128 KiB in flight) and twice the producer warps (a tile
// must be issued every ~85 ns per SM to keep up with HBM).
template <int D, bool kFp8>
struct Cfg {
    // FP8 tiles: [16 tokens][D bytes]; D = 128: 128-byte swizzled rows; D = 64: plain 64-byte rows (the tiny case:
    // its shared-memory reads are not conflict-free and need not be)
    static constexpr int kElemBytes = kFp8 ? 1 : 2;
    // one elected lane per producer warp; tiles are dealt round-robin to them (one lane is issue-rate bound)
    static constexpr int kProducerWarps = kFp8 ? 4 : COMEM_BF16_PRODUCER_WARPS;
    static constexpr int kThreads = kConsumerThreads + kProducerWarps * 32;
    // Register budgets (COMEM_K1_SETMAXNREG): the kernel is LAUNCHED with kLaunchRegs per thread, so that the small
    // combine kernel's CTAs fit beside it (384 x 144 leaves 10 240 of the SM's 65 536); the producer warpgroup then
    // shrinks to kProducerRegs and hands the difference to the two consumer warpgroups:
    // 8 x (kConsumerRegs - kLaunchRegs) <= 4 x (kLaunchRegs - kProducerRegs).
    static constexpr int kLaunchRegs = kK1LaunchRegs, kProducerRegs = 72, kConsumerRegs = 176;
    static constexpr int kPrefetch = kFp8 ? (2 * kPrefetchTiles < 32 ? 2 * kPrefetchTiles : 32) : kPrefetchTiles;
    static_assert(kPrefetch <= 32, "one prefetched tile per lane");
    static constexpr int kTileBytes = kTileTokens * D * kElemBytes;  // one K (or V) tile
    static constexpr int kStageBytes = 2 * kTileBytes;      // K + V
    // kStages % kConsumerWarps == 0 so that a ring stage always belongs to the same consumer warp:
    // a warp then never waits on a stage more than one phase ahead of the barrier (mbarrier waits
    // carry only the phase PARITY; out-of-order TMA completion could otherwise alias two phases).
    static constexpr int kStages = 128 * 1024 / kStageBytes;  // 128 KiB of K+V in flight per SM: 16 (bf16, D 128) or 32
    static constexpr int kScaleBytes = kFp8 ? kStages * 8 : 0;  // per ring stage: {k_scale, v_scale} of the tile's page
    static_assert(kStages % kConsumerWarps == 0, "ring stages must map to a fixed consumer warp");
    static constexpr int kRowPitch = D + 4;                       // floats; see S6
    static constexpr int kStateOff = kMaxGroup * kRowPitch;       // m[8], l[8], lx[8] follow the rows
    static constexpr int kScratchFloatsPerWarp = kStateOff + 3 * kMaxGroup;
    // the scratch area doubles as merge.cuh's staging area (never live at the same time)
    static constexpr int kS6ScratchBytes = kConsumerWarps * kScratchFloatsPerWarp * 4;
    static constexpr int kScratchBytes =
        kS6ScratchBytes > MergeCfg<D>::kStageBytes ? kS6ScratchBytes : MergeCfg<D>::kStageBytes;
    static constexpr int kKSteps = D / 16;  // QK^T k-steps == PV m-tiles
    static constexpr int kTilesPerPass = kFp8 ? COMEM_FP8_TILES_PER_PASS : 1;  // tiles a consumer warp takes per online-softmax update
};

// `fused`: the kernel also merges (S7) and needs merge.cuh's staging area; un-fused (the merge runs as the small
// dependent kernel of combine.cu) it leaves that shared memory free, so that kernel's CTAs fit beside this one's.
template <int D, bool kFp8>
__host__ __device__ constexpr size_t smem_bytes_for(int batch, bool fused = true)
{
    using C = Cfg<D, kFp8>;
    return 1024 /* alignment slack */ + (size_t)C::kStages * C::kStageBytes +
           (size_t)(fused ? C::kScratchBytes : C::kS6ScratchBytes) +
           (2 * C::kStages + 2) * 8 + C::kScaleBytes + ((size_t)batch + 1) * 4 + 16;
}

struct SegPos {
    int b, kvh, j, T;  // sequence, kv head, tile index within the sequence, tiles in the sequence
};

// Locate linear tile x: the b with Hkv*prefix[b] <= x < Hkv*prefix[b+1].
__device__ __forceinline__ SegPos locate(int64_t x, const int *prefix, int batch, int hkv)
{
    int lo = 0, hi = batch;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)hkv * prefix[mid] <= x) lo = mid; else hi = mid;
    }
    SegPos s;
    s.b = lo;
    s.T = prefix[lo + 1] - prefix[lo];
    const int rel = (int)(x - (int64_t)hkv * prefix[lo]);
    s.kvh = rel / s.T;
    s.j = rel - s.kvh * s.T;
    return s;
}

#ifndef COMEM_K1_SETMAXNREG
#define COMEM_K1_SETMAXNREG 1  // measured: C2 over a cold 20-step run 22.6 -> 21.0 us, steady state 19.8 -> 19.5; C3 / C4 unchanged
#endif
// kEarly: the instance that holds the early mode (launched when COMEM_LAUNCH_KV_PREFIX_IMMUTABLE is set).  The classic
// instance carries none of its tests in the tile loop: the FP8 consumers are bound by their issue slots, and the mode
// costs them 5 % on long steps (C4 with the FP8 cache, same box: 747 us with the tests compiled in, 701 without).
template <int D, bool kFp8, bool kEarly>
#if COMEM_K1_SETMAXNREG
__global__ void __maxnreg__(kK1LaunchRegs)
#else
__global__ void __launch_bounds__((Cfg<D, kFp8>::kThreads), 1)
#endif
decode_split_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v,
                    const __grid_constant__ CUtensorMap tm_kh, const __grid_constant__ CUtensorMap tm_vh,
                    const DecodeParams p)
{
    using C = Cfg<D, kFp8>;
    constexpr int kThreads = C::kThreads;
    constexpr int kProducerWarps = C::kProducerWarps;
    [[maybe_unused]] constexpr int kFp8Chunks = D / 64;  // FP8: 16-byte chunks of a K row each lane reads (S3)
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t ring = (raw + 1023u) & ~1023u;  // 1024-aligned: the 128B-swizzle atom
    uint8_t *ring_ptr = smem_raw + (ring - raw);
    float *scratch = reinterpret_cast<float *>(ring_ptr + C::kStages * C::kStageBytes);
    uint64_t *bars = reinterpret_cast<uint64_t *>(reinterpret_cast<uint8_t *>(scratch) +
                                                  (p.fuse_combine ? C::kScratchBytes : C::kS6ScratchBytes));
    const uint32_t scales0 = smem_u32(bars + 2 * C::kStages + 2);  // FP8 only: float2 per ring stage
    int *prefix = reinterpret_cast<int *>(reinterpret_cast<uint8_t *>(bars + 2 * C::kStages + 2) + C::kScaleBytes);
    const uint32_t full0 = smem_u32(bars);
    const uint32_t empty0 = full0 + 8 * C::kStages;
    const uint32_t merge_bar = empty0 + 8 * C::kStages;  // completion of merge.cuh's bulk copies
    const uint32_t verdict_bar = merge_bar + 8;          // early mode: the schedule guess has been validated (or not)

    // A CTA cuts at most two segments: its first (slot 0) and its last (slot 1; slot 0 if it has one segment only).
    // Per slot: {this CTA merges?, first record's kind, i_first, nsplit, arrival counter index, first output row}.
    __shared__ int s_seg[2][6];
    __shared__ int s_e[kAlignedMaxSegs + 1];  // segment-aligned schedule (schedule.cuh): CTAs before each segment
    __shared__ int s_aligned, s_valid;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    COMEM_STAMP(0);
#ifdef COMEM_TRACE
    if (p.trace && threadIdx.x == 0) {
        unsigned smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        p.trace[blockIdx.x * 16 + 15] = smid;
    }
#endif

    if (threadIdx.x == 0) {
        for (int s = 0; s < C::kStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 1);
        }
        mbar_init(merge_bar, 1);
        mbar_init(verdict_bar, 1);
        fence_mbar_init();
    }
    if (warp == kConsumerWarps && lane == 0) {  // first producer warp
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
        if (p.host_tier) {  // second tier: a pool in pinned host memory (block-table entries < 0), bf16 only
            tma_prefetch_desc(&tm_kh);
            tma_prefetch_desc(&tm_vh);
        }
    }
    // Nothing above touched global data.  The inputs may still be written by the kernel running
    // before this one (kv_append bumps seq_lens), so nothing read before the wait is trusted -- but
    // an L2 prefetch is a hint on a coherent cache and may run now: the small control inputs
    // (seq_lens, block table, q) are pulled from DRAM while the previous grid drains, and the
    // dependent chain seq_lens -> block table -> first TMA after the wait then runs at L2 latency.
    {
        const int64_t gtid = (int64_t)blockIdx.x * kThreads + threadIdx.x;
        if (gtid < (((int64_t)p.batch * 4 + 127) >> 7))
            prefetch_l2(reinterpret_cast<const char *>(p.seq_lens) + (gtid << 7));
        if (gtid < (((int64_t)p.batch * p.max_pages * 4 + 127) >> 7))
            prefetch_l2(reinterpret_cast<const char *>(p.block_table) + (gtid << 7));
        if (gtid < (((int64_t)p.batch * p.num_q_heads * D * 2 + 127) >> 7))
            prefetch_l2(reinterpret_cast<const char *>(p.q) + (gtid << 7));
    }
    // S1, the schedule: everything below is a function of seq_lens (and the launch dimensions).
    // It is computed SPECULATIVELY before griddepcontrol.wait, from whatever seq_lens holds while the
    // previous kernel may still be running (it may be kv_append, about to bump every length), and
    // validated after the wait by re-reading seq_lens: a decode step changes a sequence's tile count
    // once in 16 steps, so the guess is nearly always right and the ~2 us of cold, division-heavy
    // schedule code run under the previous kernel's tail instead of on this launch's critical path.
    // A wrong guess just runs the same code again.  seq_lens is read with ld.cg (L2) throughout, so
    // no stale copy can sit in L1.
    int64_t total = 0, c0 = 0, c1 = 0;
    int nc = 0, al_first = 0, al_count = 0;  // aligned: first CTA and CTA count of this CTA's segment
    bool aligned = false;
    const int cta = blockIdx.x;
    // (COMEM_DEBUG_STALE_GUESS=1, a testing aid: the FIRST schedule is computed from lengths 16 tokens short, as if the
    // append kernel had not run yet, so that the validation fails and the recovery paths run on every launch)
    int guess_bias = p.debug_stale_guess ? kTileTokens : 0;
    auto guess_len = [&](int L) { return L > guess_bias ? L - guess_bias : L; };
    auto compute_schedule = [&]() {
        // exclusive prefix of tiles per sequence (warp 0); kept small: no unrolling
        if (warp == 0) {
            if (p.batch <= 32) {
#ifdef COMEM_TRACE
                if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 11] = globaltimer_ns();
#endif
                const int mine = lane < p.batch ? seq_tiles(guess_len(__ldcg(p.seq_lens + lane)), p.window, p.sinks) : 0;
                int incl = mine;
#ifdef COMEM_TRACE
                if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 12] = globaltimer_ns() + (mine == -12345);
#endif
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(kFull, incl, o);
                    if (lane >= o) incl += v;
                }
                if (lane < p.batch) prefix[lane] = incl - mine;
                if (lane == 31) prefix[p.batch] = incl;
            } else {
                const int per = (p.batch + 31) >> 5;
                const int b0 = lane * per;
                int sum = 0;
#pragma unroll 1
                for (int i = 0; i < per; ++i)
                    if (b0 + i < p.batch) sum += seq_tiles(guess_len(__ldcg(p.seq_lens + b0 + i)), p.window, p.sinks);
                int incl = sum;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(kFull, incl, o);
                    if (lane >= o) incl += v;
                }
                int run = incl - sum;
#pragma unroll 1
                for (int i = 0; i < per; ++i)
                    if (b0 + i < p.batch) {
                        prefix[b0 + i] = run;
                        run += seq_tiles(guess_len(__ldcg(p.seq_lens + b0 + i)), p.window, p.sinks);
                    }
                if (lane == 31) prefix[p.batch] = incl;
            }
            // Few long segments?  Then deal whole CTAs to segments (schedule.cuh, "segment-aligned
            // variant"; the same arithmetic as aligned_build, two segments per lane).
            __syncwarp();
            const int S = p.batch * p.num_kv_heads;
            const int64_t tot = (int64_t)p.num_kv_heads * prefix[p.batch];
            bool ok = S <= kAlignedMaxSegs && tot >= (int64_t)gridDim.x * kMinTilesPerCta;
            if (ok) {  // warp-uniform
                const int ideal = ideal_tiles_per_cta(tot, (int)gridDim.x);
                bool mine_ok = true;
                for (int sidx = lane; sidx < S; sidx += 32) {
                    const int b = sidx / p.num_kv_heads, kvh = sidx - b * p.num_kv_heads;
                    const int T = prefix[b + 1] - prefix[b];
                    const int64_t before = (int64_t)p.num_kv_heads * prefix[b] + (int64_t)kvh * T;
                    const int e_lo = aligned_boundary(before, tot, (int)gridDim.x);
                    const int e_hi = aligned_boundary(before + T, tot, (int)gridDim.x);
                    s_e[sidx + 1] = e_hi;
                    mine_ok = mine_ok && aligned_segment_ok(T, e_hi - e_lo, ideal);
                }
                if (lane == 0) s_e[0] = 0;
                ok = __all_sync(kFull, mine_ok);
            }
            if (lane == 0) s_aligned = ok ? 1 : 0;
        }
        __syncthreads();
#ifdef COMEM_TRACE
        if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 13] = globaltimer_ns();
#endif
        // this CTA's range [c0, c1) of the linearised tile space
        total = (int64_t)p.num_kv_heads * prefix[p.batch];
        aligned = s_aligned != 0;
        c0 = c1 = 0;
        if (total == 0) return;
        if (aligned) {
            nc = (int)gridDim.x;
            int lo = 0, hi = p.batch * p.num_kv_heads;  // s_e[lo] <= cta < s_e[hi]
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (s_e[mid] <= cta) lo = mid; else hi = mid;
            }
            const int b = lo / p.num_kv_heads, kvh = lo - b * p.num_kv_heads;
            const int T = prefix[b + 1] - prefix[b];
            const int64_t seg0 = (int64_t)p.num_kv_heads * prefix[b] + (int64_t)kvh * T;
            al_first = s_e[lo];
            al_count = s_e[lo + 1] - al_first;
            c0 = aligned_cta_begin(seg0, T, cta - al_first, al_count);
            c1 = aligned_cta_begin(seg0, T, cta - al_first + 1, al_count);
        } else {
            nc = sched_num_ctas(total, (int)gridDim.x);
            if (cta < nc) {
                c0 = cta_begin(cta, total, nc);
                c1 = cta_begin(cta + 1, total, nc);
            }
        }
    };
    compute_schedule();  // speculative
    guess_bias = 0;        // (any later call computes the real schedule)
    // EARLY MODE (COMEM_LAUNCH_KV_PREFIX_IMMUTABLE, p.kv_immutable): the caller has PROMISED that nothing still running
    // writes the cached rows below each sequence's last tile, their block-table entries or their page scales.  Then
    // this CTA does not sit in griddepcontrol.wait while the previous kernel drains: its producers stream those tiles
    // NOW, from the guessed schedule, and -- with COMEM_LAUNCH_Q_STABLE (q is not being written either) -- its consumers
    // fold them as they land.  The wait moves to the first point where the CTA needs something the previous kernel may
    // still write or must not yet see written: a sequence's LAST tile (the append kernel's row), seq_lens itself, and
    // any global store (S6).  That point is CTA-local tile index X: the sequence-last tile if the CTA's first segment
    // portion ends with it, else the end of that portion (= the end of the CTA's range).  There, one producer warp
    // waits for the previous grid, re-reads seq_lens, compares the tile counts with the guess and publishes the
    // verdict on an mbarrier; everybody else picks it up when they get to X.  A wrong guess (a length crossed a tile
    // boundary: once in 16 decode steps per sequence) aborts the attempt: what was streamed is dropped, the barriers
    // are re-initialised and the CTA runs again in the classic order below.  Bits are the same in both modes: the
    // schedule, the tile -> warp map and every reduction order are unchanged.
    bool early = kEarly && p.kv_immutable != 0 && p.window <= 0 && c0 < c1;
    __shared__ int s_abort;
    if (!early) {
        // Classic order.  Still before the wait: ask the TMA unit to pull this CTA's first tiles into L2.  Cached KV
        // rows of old tokens are immutable, so a prefetch from the guessed schedule and the block table as it reads
        // now is at worst useless (the page index is clamped to the table row, a bad page id is an out-of-range
        // tensor coordinate: both harmless for a hint).  HBM is idle while the previous kernel drains its tail; the
        // first real loads after the wait then hit L2.
        if (warp == kConsumerWarps && c0 < c1 && p.window <= 0) {  // (identity tile map only)
            const SegPos sp = locate(c0, prefix, p.batch, p.num_kv_heads);
            const int64_t rem = c1 - c0;
            int cnt = (int)(rem < (int64_t)(sp.T - sp.j) ? rem : (int64_t)(sp.T - sp.j));
            cnt = cnt < C::kPrefetch ? cnt : C::kPrefetch;
            if (lane < cnt) {
                const int jj = sp.j + lane;
                int page = jj >> p.page_tile_shift;
                page = page < p.max_pages ? page : p.max_pages - 1;
                const int pid = __ldcg(p.block_table + (int64_t)sp.b * p.max_pages + page);
                const int slot0 = (jj & ((1 << p.page_tile_shift) - 1)) << kTileShift;
                // tensor coordinates of the tile: {d, token row, -, kv head}, or {d, slot, kv head, page} for the HND layout
                const int c1 = (kFp8 && p.kv_hnd) ? slot0 : pid * p.page_size + slot0;
                const int c2 = (kFp8 && p.kv_hnd) ? sp.kvh : 0, c3 = (kFp8 && p.kv_hnd) ? pid : sp.kvh;
                if (pid >= 0) {  // (a host-tier page is not worth a hint: it would cross the host link twice)
                    tma_prefetch_tile_4d(&tm_k, 0, c1, c2, c3);
                    tma_prefetch_tile_4d(&tm_v, 0, c1, c2, c3);
                }
            }
        }
        pdl_wait_prior_grid();
        COMEM_STAMP(1);
        if (warp == 0) {  // validate the guess against the lengths as they are now
            bool same = true;
#pragma unroll 1
            for (int b = lane; b < p.batch; b += 32)
                same = same && seq_tiles(__ldcg(p.seq_lens + b), p.window, p.sinks) == prefix[b + 1] - prefix[b];
            same = __all_sync(kFull, same);
            if (lane == 0) s_valid = same ? 1 : 0;
        }
#ifdef COMEM_TRACE
        if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 11] = globaltimer_ns();
        if (p.trace && threadIdx.x == kConsumerThreads) p.trace[blockIdx.x * 16 + 12] = globaltimer_ns();
        if (p.trace && threadIdx.x == 32) p.trace[blockIdx.x * 16 + 13] = globaltimer_ns();
#endif
        __syncthreads();
        if (!s_valid) {
            __syncthreads();  // everyone has read s_valid and the old tables before warp 0 rewrites them
            compute_schedule();
        }
    }
    pdl_launch_dependents();
    COMEM_STAMP(2);

    // One pass, or two when an early attempt is aborted.  The attempt loop is written once per role (producers,
    // consumers) so that each role's register budget (setmaxnreg, below) dominates its own code.
    // S8: rows of empty sequences (reading R9): +0.0 and lse = -inf, dealt round-robin to the CTAs.
    auto write_empty_rows = [&]() {
        if (!p.fuse_combine) return;
        for (int b = blockIdx.x; b < p.batch; b += gridDim.x) {
            if (prefix[b + 1] != prefix[b]) continue;
            const int64_t row0 = (int64_t)b * p.num_q_heads;
            for (int e = threadIdx.x; e < p.num_q_heads * D; e += kThreads) p.out[row0 * D + e] = __float2bfloat16_rn(0.f);
            if (p.lse_out)
                for (int h = threadIdx.x; h < p.num_q_heads; h += kThreads) p.lse_out[row0 + h] = -INFINITY;
        }
    };
    // early mode: CTA-local index of the first tile that needs the wait (producers: xp, consumers: xc)
    int xp = 0, xc = 0;
    bool early_pending = false, aborted = false;
    // start of an attempt; false: this CTA has nothing to stream
    auto attempt_begin = [&]() -> bool {
    if (!early) {
        write_empty_rows();
        if (c0 >= c1) return false;  // nothing to stream (no tiles at all, or more CTAs than the schedule uses)
    }
    xp = xc = 0;
    if (early) {
        const SegPos sp = locate(c0, prefix, p.batch, p.num_kv_heads);
        const int64_t rem = c1 - c0;
        const int cnt0 = (int)(rem < (int64_t)(sp.T - sp.j) ? rem : (int64_t)(sp.T - sp.j));
        const int x_wait = (sp.j + cnt0 == sp.T) ? cnt0 - 1 : cnt0;
        // without COMEM_LAUNCH_Q_STABLE the consumers cannot start before the wait: the producers fill the ring once
        // (no stage is reused, so they never block on the consumers) and ask for the verdict
        xc = p.q_stable ? x_wait : 0;
        xp = p.q_stable ? x_wait : (x_wait < C::kStages ? x_wait : C::kStages);
    }
    early_pending = early;
    aborted = false;
    return true;
    };
    // end of an attempt; true: the early attempt was aborted, run again in the classic order
    auto attempt_end = [&]() -> bool {
    if (!early) return false;
    // End of an early attempt: all threads meet; either it went through (the empty rows are still to write: global
    // stores, so after the wait every thread has passed by now), or the guess was wrong and the CTA starts over in
    // the classic order with fresh barriers and the real schedule.
    __syncthreads();
    if (*reinterpret_cast<volatile int *>(&s_abort) == 0) {
        write_empty_rows();
        return false;
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < C::kStages; ++s) {
            mbar_inval(full0 + 8 * s);
            mbar_inval(empty0 + 8 * s);
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 1);
        }
        mbar_inval(merge_bar);
        mbar_init(merge_bar, 1);
        fence_mbar_init();
    }
    compute_schedule();  // (its barrier also publishes the fresh mbarriers)
    early = false;
    return true;
    };

    if (warp >= kConsumerWarps) {
#if COMEM_K1_SETMAXNREG
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::kProducerRegs));
#endif
      do {
        if (!attempt_begin()) return;
        // ------------------------------ S2: page-gather producers -----------------------------
        // Producer warp pw issues the CTA's tiles with (CTA-local index) % kProducerWarps == pw; tile
        // tl always lands in ring stage tl % kStages, in the ring's pass number tl / kStages.
        static_assert((C::kStages & (C::kStages - 1)) == 0 && C::kStages % kProducerWarps == 0, "ring indexing");
        static_assert((kProducerWarps & (kProducerWarps - 1)) == 0, "round-robin by mask");
        constexpr int kStageShift = (C::kStages == 16) ? 4 : (C::kStages == 32 ? 5 : 6);
        static_assert((1 << kStageShift) == C::kStages, "kStageShift");
        const int pw = warp - kConsumerWarps;
        // K/V bytes are used once per step: evict-first keeps them from displacing the L2-resident
        // control data, partial records and whatever else the model keeps there between steps
        const uint64_t stream_policy = l2_policy_evict_first();
        const int tiles_per_page_mask = (1 << p.page_tile_shift) - 1;
        int tl0 = 0;  // CTA-local index of the current segment's first tile
        int64_t x = c0;
        // Early mode: the wait, the validation of the guessed schedule and the verdict (see above).  Producer warp 0
        // decides, the others read its verdict.
        auto verdict = [&]() {
            if (pw == 0) {
                pdl_wait_prior_grid();
                bool same = true;
#pragma unroll 1
                for (int b = lane; b < p.batch; b += 32)
                    same = same && seq_tiles(__ldcg(p.seq_lens + b), p.window, p.sinks) == prefix[b + 1] - prefix[b];
                same = __all_sync(kFull, same);
                if (lane == 0) {
                    *reinterpret_cast<volatile int *>(&s_abort) = same ? 0 : 1;
                    mbar_arrive(verdict_bar);  // release: s_abort is visible to whoever waits on the barrier
                }
                aborted = !same;
            } else {
                mbar_wait(verdict_bar, 0u);
                pdl_wait_prior_grid();
                aborted = *reinterpret_cast<volatile int *>(&s_abort) != 0;
            }
            early_pending = false;
#ifdef COMEM_TRACE
            if (p.trace && threadIdx.x == kConsumerThreads) p.trace[blockIdx.x * 16 + 14] = globaltimer_ns();
#endif
        };
        while (x < c1 && !(kEarly && aborted)) {
            const SegPos sp = locate(x, prefix, p.batch, p.num_kv_heads);
            const int64_t rem = c1 - x;
            const int cnt = (int)(rem < (int64_t)(sp.T - sp.j) ? rem : (int64_t)(sp.T - sp.j));
            const int32_t *bt = p.block_table + (int64_t)sp.b * p.max_pages;
            // sequence tile index -> logical tile (identity unless a sliding window is set)
            const WinTiles wt = win_tiles(p.window > 0 ? __ldcg(p.seq_lens + sp.b) : 0, p.window, p.sinks);
            // issue the segment's tiles [lo, hi) (indices within this CTA's portion of the segment)
            auto issue_range = [&](const int lo, const int hi) {
                // The per-tile metadata (block-table entry, then -- FP8 -- the page's two scales, which depend on it)
                // is fetched 32 tiles at a time, one tile per lane, and kept TWO batches ahead of the tiles being
                // issued: a batch's loads are in flight while the previous batches' TMAs are issued, so the dependent
                // round trips to L2 / DRAM never stop the issue loop (they did: half of the producers' samples).
                auto load_pid = [&](int base) -> int {
                    if (base + lane >= hi) return 0;
                    return __ldg(bt + (win_logical_tile(wt, sp.j + base + lane) >> p.page_tile_shift));
                };
                auto load_scales = [&](int base, int pid, float &ks, float &vs) {
                    ks = vs = 0.f;
                    if constexpr (kFp8) {
                        if (base + lane < hi) {
                            ks = __ldg(p.k_scale + (int64_t)pid * p.num_kv_heads + sp.kvh);
                            vs = __ldg(p.v_scale + (int64_t)pid * p.num_kv_heads + sp.kvh);
                        }
                    }
                };
                // (bf16: one L2-latency load per 32 tiles of 8 KiB is covered by the ring, and a short CTA -- config 2
                // has ~110 tiles -- is better off with the shortest path to its first TMA: measured, so not pipelined.)
                constexpr bool kMetaAhead = kFp8;
                int pid = kMetaAhead ? load_pid(lo) : 0, pid_next = kMetaAhead ? load_pid(lo + 32) : 0;
                float ks = 0.f, vs = 0.f;  // FP8: the page's scales for this kv head
                if constexpr (kMetaAhead) load_scales(lo, pid, ks, vs);
                for (int base = lo; base < hi; base += 32) {
                    float ks_next = 0.f, vs_next = 0.f;
                    int pid_next2 = 0;
                    if constexpr (kMetaAhead) {
                        load_scales(base + 32, pid_next, ks_next, vs_next);
                        pid_next2 = load_pid(base + 64);
                    } else {
                        pid = load_pid(base);
                    }
                    const int jj = win_logical_tile(wt, sp.j + base + lane);
                    const int m = hi - base < 32 ? hi - base : 32;
                    for (int i = (pw - (tl0 + base)) & (kProducerWarps - 1); i < m; i += kProducerWarps) {
                        const int tl = tl0 + base + i;
                        const int stage = tl & (C::kStages - 1);
                        const uint32_t phase = (uint32_t)(tl >> kStageShift) & 1u;
                        mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                        const int pid_i = __shfl_sync(kFull, pid, i);
                        const int jj_i = __shfl_sync(kFull, jj, i);
                        float ks_i = 0.f, vs_i = 0.f;
                        if constexpr (kFp8) {
                            ks_i = __shfl_sync(kFull, ks, i);
                            vs_i = __shfl_sync(kFull, vs, i);
                        }
                        if (elect_one()) {  // (not `lane == 0`: see elect_one)
                            const int slot0 = (jj_i & tiles_per_page_mask) << kTileShift;
                            // block-table entry e >= 0: page e of the device pool; e < 0: page -1 - e of the host tier
                            const bool host_page = !kFp8 && pid_i < 0;
                            const int pg = host_page ? -1 - pid_i : pid_i;
                            const CUtensorMap *mk = host_page ? &tm_kh : &tm_k, *mv = host_page ? &tm_vh : &tm_v;
                            const int c1 = (kFp8 && p.kv_hnd) ? slot0 : pg * p.page_size + slot0;
                            const int c2 = (kFp8 && p.kv_hnd) ? sp.kvh : 0, c3 = (kFp8 && p.kv_hnd) ? pg : sp.kvh;
                            const uint32_t dst = ring + stage * C::kStageBytes;
                            const uint32_t bar = full0 + 8 * stage;
                            if constexpr (kFp8)  // ordered before the consumers' wait by the arrive below (release) and their wait (acquire)
                                asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(scales0 + 8 * stage), "f"(ks_i), "f"(vs_i) : "memory");
                            mbar_arrive_expect_tx(bar, C::kStageBytes);
                            tma_load_4d_hint(dst, mk, bar, 0, c1, c2, c3, stream_policy);
                            tma_load_4d_hint(dst + C::kTileBytes, mv, bar, 0, c1, c2, c3, stream_policy);
                        }
                    }
                    pid = pid_next;
                    pid_next = pid_next2;
                    ks = ks_next;
                    vs = vs_next;
                }
            };
            int lo = 0;
            if (kEarly && early_pending) {  // (first segment only: xp lies inside it)
                lo = xp - tl0 < cnt ? xp - tl0 : cnt;
                issue_range(0, lo);
                verdict();
                if (kEarly && aborted) break;
            }
            issue_range(lo, cnt);
            x += cnt;
            tl0 += cnt;
        }
      } while (attempt_end());
    } else {
#if COMEM_K1_SETMAXNREG
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::kConsumerRegs));
#endif
    do {
    if (!attempt_begin()) return;
    // ------------------------------ consumers: S3..S6 -----------------------------------------
    const int quad = lane >> 2;  // score row = query head within the group
    const int qlane = lane & 3;
    // ldmatrix lane addressing inside a tile: matrix (lane / 8), row (lane % 8)
    const int ld_mat = lane >> 3;
    const int ld_tok = ((ld_mat >> 1) << 3) + (lane & 7);
    const uint32_t ld_row_off = ld_tok * 128;
    const uint32_t ld_xor = ld_tok & 7;
    const uint32_t ld_half = ld_mat & 1;

    float *my_scratch = scratch + warp * C::kScratchFloatsPerWarp;

    uint32_t merge_phase = 0;
    bool pending_first = false;  // slot 0's ticket was taken in mid-stream; its outcome is in s_seg[0][0]

    // S7: publish the stored partial, take a ticket on the segment's arrival counter; the CTA that
    // arrives LAST on a segment merges all of that segment's partials and re-arms the counter.
    // release = fence + relaxed ticket (cumulative over a barrier: the whole CTA's partial stores
    // happen-before the ticket); acquire = ticket + fence, paid only by a CTA that merges.
    // `have_first`: slot 0's ticket was already taken in mid-stream (see the segment loop); if it
    // turned out to be the last one, its merge is done here too.
    auto publish_and_merge = [&](bool have_first, bool do_cur, int cur_slot) {
        fence_proxy_async_smem();             // scratch (generic writes in S6) is the merge's TMA landing area
        named_bar_sync(1, kConsumerThreads);  // every consumer's partial stores are issued
        COMEM_STAMP(5);
        if (threadIdx.x == 0) {
            int last1 = 0;
            if (do_cur) {
                int *ctr = p.seg_counters + s_seg[cur_slot][4];
                fence_acq_rel_gpu();
                last1 = atomicAdd(ctr, 1) == s_seg[cur_slot][3] - 1;
                if (last1) *ctr = 0;  // re-armed for the next launch (ordered by the kernel boundary)
                s_seg[cur_slot][0] = last1;
            }
            if (last1 || (have_first && s_seg[0][0])) fence_acq_rel_gpu();
        }
        named_bar_sync(1, kConsumerThreads);
        COMEM_STAMP(6);
        if (have_first && s_seg[0][0]) {
            merge_partials<D>(p, warp, lane, s_seg[0][1], s_seg[0][2], s_seg[0][3], (int64_t)s_seg[0][5], scratch,
                              merge_bar, merge_phase);
            if (do_cur) named_bar_sync(1, kConsumerThreads);  // the staging area is reused below
        }
        if (do_cur && s_seg[cur_slot][0])
            merge_partials<D>(p, warp, lane, s_seg[cur_slot][1], s_seg[cur_slot][2], s_seg[cur_slot][3],
                              (int64_t)s_seg[cur_slot][5], scratch, merge_bar, merge_phase);
    };
    // early mode: pick up the producers' verdict (the previous grid has completed, the guessed schedule holds or not)
    auto need_verdict = [&]() {
        mbar_wait(verdict_bar, 0u);
        pdl_wait_prior_grid();
        aborted = *reinterpret_cast<volatile int *>(&s_abort) != 0;
        early_pending = false;
        COMEM_STAMP(1);
    };
    int64_t x = c0;
    int n = 0;        // CTA-local index of the segment's first tile
    int t = warp;     // this warp's next tile (CTA-local index)
    int stage = warp; // == t % kStages (kStages > kConsumerWarps)
    uint32_t phase = 0;

    while (x < c1) {
        if (kEarly && early_pending && xc <= n) {  // nothing of this segment may be touched before the wait (q included)
            need_verdict();
            if (kEarly && aborted) break;
        }
        const SegPos sp = locate(x, prefix, p.batch, p.num_kv_heads);
        const int64_t rem = c1 - x;
        const int cnt = (int)(rem < (int64_t)(sp.T - sp.j) ? rem : (int64_t)(sp.T - sp.j));
        const bool whole_segment = (sp.j == 0 && cnt == sp.T);
        if (!whole_segment && p.fuse_combine && threadIdx.x == 0) {
            // which CTAs cut this segment (64-bit divisions: done now, under the streaming, not in the tail)
            int *sg = s_seg[x == c0 ? 0 : 1];
            if (aligned) {
                sg[1] = 0;
                sg[2] = al_first;
                sg[3] = al_count;
            } else {
                const int64_t seg0 = x - sp.j, seg1 = seg0 + sp.T;
                const int i_first = cta_of_tile(seg0, total, nc);
                sg[1] = cta_begin(i_first, total, nc) < seg0 ? 1 : 0;  // record kind of the segment's first split
                sg[2] = i_first;
                sg[3] = cta_of_tile(seg1 - 1, total, nc) - i_first + 1;
            }
            sg[4] = sp.b * p.num_kv_heads + sp.kvh;
            sg[5] = sp.b * p.num_q_heads + sp.kvh * p.group;
        }
        // (early mode, before the verdict: possibly the length before the append -- it only decides the mask of the
        // sequence's last tile, which is not touched until the verdict is in and the length re-read)
        int seq_len = __ldcg(p.seq_lens + sp.b);
        WinTiles wt = win_tiles(seq_len, p.window, p.sinks);
        const int head0 = sp.kvh * p.group;

        // Q fragments (A operand of S = Q K^T): row = head `quad`, rows 8..15 are zero padding.
        uint32_t qf[C::kKSteps][2];
        {
            const uint32_t *qrow = reinterpret_cast<const uint32_t *>(
                p.q + ((int64_t)sp.b * p.num_q_heads + head0 + quad) * D);
            const bool live = quad < p.group;
            if constexpr (kFp8) {
                // E4M3 widens exactly to fp16, so the tensor op runs in fp16 and q is converted once per
                // segment.  The contraction index is permuted to suit 16-byte shared-memory reads of K
                // (see S3): k-step 4c + w of lane qlane covers d = 16 (2 qlane + c) + 4 w + {0,1 | 2,3}
                // (D = 64: one chunk per lane, d = 16 qlane + 4 w + ...).
#pragma unroll
                for (int c = 0; c < kFp8Chunks; ++c)
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        const int i32 = 8 * (kFp8Chunks * qlane + c) + 2 * w;
                        qf[4 * c + w][0] = live ? bf16x2_to_f16x2(__ldg(qrow + i32)) : 0u;
                        qf[4 * c + w][1] = live ? bf16x2_to_f16x2(__ldg(qrow + i32 + 1)) : 0u;
                    }
            } else {
#pragma unroll
                for (int kk = 0; kk < C::kKSteps; ++kk) {
                    qf[kk][0] = live ? __ldg(qrow + 8 * kk + qlane) : 0u;
                    qf[kk][1] = live ? __ldg(qrow + 8 * kk + 4 + qlane) : 0u;
                }
            }
        }

        float m_run = -INFINITY;  // running max (log2 domain) of head `quad`
        float l_run = 0.f;        // this thread's share of the running sum of the bf16-ROUNDED p (normaliser)
        float lx_run = 0.f;       // same for the unrounded p (only feeds lse_out)
        // FP8 cache: acc is kept in units of 2^(eref - 127 - kFp8PShift), eref = the largest biased exponent of a
        // page's v_scale seen so far (warp-uniform); see S4
        [[maybe_unused]] int eref = 0;
        float acc[C::kKSteps][4]; // O^T: rows d = 16*mt + quad (+8), cols heads 2*qlane (+1)
#pragma unroll
        for (int mt = 0; mt < C::kKSteps; ++mt) acc[mt][0] = acc[mt][1] = acc[mt][2] = acc[mt][3] = 0.f;

        // One pass of S3..S5 over NT of this warp's tiles (t, t + 8, ...) with ONE online-softmax update for all of
        // them.  NT = 2 (FP8 cache) gives the warp two independent load -> convert -> MMA chains to interleave:
        // with half the bytes per tile, a single chain per warp is latency-bound below the HBM rate.
        auto tiles_pass = [&](auto nt_tag) {
            constexpr int NT = decltype(nt_tag)::value;
            if (kEarly && early_pending && t + (NT - 1) * kConsumerWarps >= xc) {
                need_verdict();
                if (kEarly && aborted) return;
                seq_len = __ldcg(p.seq_lens + sp.b);
                wt = win_tiles(seq_len, p.window, p.sinks);
            }
            uint32_t k_base[NT], v_base[NT];
            unsigned alive[NT];
            int stg[NT];
            {
                int sg = stage;
                uint32_t ph = phase;
#pragma unroll
                for (int k = 0; k < NT; ++k) {
                    mbar_wait(full0 + 8 * sg, ph);
                    stg[k] = sg;
                    k_base[k] = ring + sg * C::kStageBytes;
                    v_base[k] = k_base[k] + C::kTileBytes;
                    // which of the tile's 16 tokens count: all but the ones past seq_len (last tile) and, under a
                    // sliding window, the ones in the gap between the sinks and the window
                    alive[k] = win_alive_mask(wt, seq_len, win_logical_tile(wt, sp.j + (t + k * kConsumerWarps - n)));
                    sg += kConsumerWarps;
                    if (sg >= C::kStages) {
                        sg -= C::kStages;
                        ph ^= 1u;
                    }
                }
            }
#ifdef COMEM_TRACE
            if (t == 0) COMEM_STAMP(3);
#endif

            // S3: scores for 2 n-tiles of 8 tokens per tile
            float s[NT][2][4];
            float sl2[NT], v_scale[NT];
#pragma unroll
            for (int k = 0; k < NT; ++k) {
#pragma unroll
                for (int j = 0; j < 4; ++j) s[k][0][j] = s[k][1][j] = 0.f;
                sl2[k] = p.scale_log2;
                v_scale[k] = 1.f;
            }
            if constexpr (kFp8) {
                // The tile is [16 tokens][128 B], 128-byte swizzled.  Lane (quad, qlane) reads, of token rows
                // row0 and row0 + 2 (below), the 16-byte chunks 2 qlane and 2 qlane + 1: a quarter-warp (two rows that
                // differ in bit 0, even chunks ^ row) touches every bank once.  Each 32-bit word is one k-step's
                // B fragment: bytes 0,1 -> b0, bytes 2,3 -> b1 (the permutation q was loaded with).
#pragma unroll
                for (int k = 0; k < NT; ++k) {
                    float2 sc;
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(sc.x), "=f"(sc.y) : "r"(scales0 + 8 * stg[k]));
                    sl2[k] *= sc.x;
                    v_scale[k] = sc.y;
                }
#pragma unroll
                for (int c = 0; c < kFp8Chunks; ++c) {
                    // Score column `quad` of n-tile 0 is token row0 = 4 (quad / 2) + quad % 2 and of n-tile 1 token
                    // row0 + 2, so that a lane's four scores are the CONSECUTIVE tokens 4 qlane .. 4 qlane + 3: the
                    // token order in which ldmatrix.trans.b8 hands out V (S5).
                    const uint32_t chunk = (uint32_t)(kFp8Chunks * qlane + c);
                    const int row0 = 4 * (quad >> 1) + (quad & 1);
                    const uint32_t off0 = (D == 128 ? (chunk ^ (uint32_t)(row0 & 7)) : chunk) << 4;
                    const uint32_t off1 = (D == 128 ? (chunk ^ (uint32_t)((row0 + 2) & 7)) : chunk) << 4;
#pragma unroll
                    for (int k = 0; k < NT; ++k) {
                        const uint4 ka = lds128(k_base[k] + row0 * D + off0), kb = lds128(k_base[k] + (row0 + 2) * D + off1);
                        const uint32_t wa[4] = {ka.x, ka.y, ka.z, ka.w}, wb[4] = {kb.x, kb.y, kb.z, kb.w};
#pragma unroll
                        for (int w = 0; w < 4; ++w) {
                            const int kk = 4 * c + w;
                            mma_f16_16816(s[k][0], qf[kk][0], 0u, qf[kk][1], 0u, e4m3x2_lo_to_f16x2(wa[w]), e4m3x2_hi_to_f16x2(wa[w]));
                            mma_f16_16816(s[k][1], qf[kk][0], 0u, qf[kk][1], 0u, e4m3x2_lo_to_f16x2(wb[w]), e4m3x2_hi_to_f16x2(wb[w]));
                        }
                    }
                }
            } else {
#pragma unroll
                for (int kk = 0; kk < C::kKSteps; ++kk) {
#pragma unroll
                    for (int k = 0; k < NT; ++k) {
                        uint32_t kf[4];
                        const uint32_t chunk = ((2 * kk) & 7) | ld_half;
                        ldmatrix_x4(kf, k_base[k] + (kk >> 2) * 2048 + ld_row_off + ((chunk ^ ld_xor) << 4));
                        mma_bf16_16816(s[k][0], qf[kk][0], 0u, qf[kk][1], 0u, kf[0], kf[1]);
                        mma_bf16_16816(s[k][1], qf[kk][0], 0u, qf[kk][1], 0u, kf[2], kf[3]);
                    }
                }
            }
            float sv[NT][4];  // tokens 2q, 2q+1, 2q+8, 2q+9 (FP8: 4q .. 4q+3) of head `quad`
#pragma unroll
            for (int k = 0; k < NT; ++k) {
                sv[k][0] = s[k][0][0] * sl2[k];
                sv[k][1] = s[k][0][1] * sl2[k];
                sv[k][2] = s[k][1][0] * sl2[k];
                sv[k][3] = s[k][1][1] * sl2[k];
                if (alive[k] != 0xffffu) {
                    // edge tile: mask by index (never by arithmetic) and zero the dead V rows so that
                    // NaN/Inf garbage in tokens that do not count cannot reach the accumulators (0 * NaN).
                    // this lane's four scores: tokens 2q, 2q+1, 2q+8, 2q+9 (bf16) or 4q .. 4q+3 (FP8, see S3)
                    const int tok = kFp8 ? 4 * qlane : 2 * qlane;
                    constexpr int kSecond = kFp8 ? 2 : 8;
                    if (!((alive[k] >> tok) & 1u)) sv[k][0] = -INFINITY;
                    if (!((alive[k] >> (tok + 1)) & 1u)) sv[k][1] = -INFINITY;
                    if (!((alive[k] >> (tok + kSecond)) & 1u)) sv[k][2] = -INFINITY;
                    if (!((alive[k] >> (tok + kSecond + 1)) & 1u)) sv[k][3] = -INFINITY;
                    constexpr int kChunksPerRow = D * C::kElemBytes / 16;  // 16-byte chunks per V row
                    for (int idx = lane; idx < kTileTokens * kChunksPerRow; idx += 32) {
                        const int row = idx / kChunksPerRow;
                        if ((alive[k] >> row) & 1u) continue;
                        const int ch = idx % kChunksPerRow;
                        const uint32_t a = (kFp8 && D == 64) ? v_base[k] + row * 64 + (ch << 4)
                                                             : v_base[k] + (ch >> 3) * 2048 + row * 128 + ((ch & 7) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(a), "r"(0u) : "memory");
                    }
                    fence_proxy_async_smem();
                    __syncwarp();
                }
            }

            // S4: online softmax for head `quad` over these tiles' tokens
            float tmax = fmaxf(fmaxf(sv[0][0], sv[0][1]), fmaxf(sv[0][2], sv[0][3]));
#pragma unroll
            for (int k = 1; k < NT; ++k) tmax = fmaxf(tmax, fmaxf(fmaxf(sv[k][0], sv[k][1]), fmaxf(sv[k][2], sv[k][3])));
            tmax = fmaxf(tmax, __shfl_xor_sync(kFull, tmax, 1));
            tmax = fmaxf(tmax, __shfl_xor_sync(kFull, tmax, 2));
            const float m_new = fmaxf(m_run, tmax);
            const float alpha = ex2(m_run - m_new);
            m_run = m_new;
            uint32_t p01[NT], p23[NT];
            float esum = 0.f;
            [[maybe_unused]] float rsum = 0.f;
            // FP8 cache: the page's v_scale = f * 2^ev rides on p, which the tensor op wants in fp16.  p <= 1 times a
            // scale of ~1e-3 would sit in the fp16 SUBNORMALS (below 2^-14) for every token more than a few nats under
            // the row maximum and lose its bits while l still counts it.  So only f * 2^(ev - eref) goes on p, lifted
            // by 2^kFp8PShift to the top of the fp16 range (p' < 2^15, normal down to e = 2^-(14 + kFp8PShift)), with
            // eref the running maximum of ev: when a page with a larger exponent arrives, acc is multiplied by the
            // exact power of two beta = 2^(eref_old - eref_new), like alpha for the running softmax maximum.  S6
            // multiplies the finished accumulator by 2^(eref - 127 - kFp8PShift).  A zero / subnormal scale counts as 0.
            [[maybe_unused]] float pscale[NT];
            float beta = 1.f;
            if constexpr (kFp8) {
                int ev[NT], emax = eref;
#pragma unroll
                for (int k = 0; k < NT; ++k) {
                    ev[k] = (int)((__float_as_uint(v_scale[k]) >> 23) & 0xffu);
                    emax = max(emax, ev[k]);
                }
                if (emax != eref) {
                    const int sh = 127 + eref - emax;
                    beta = sh > 0 ? __uint_as_float((uint32_t)sh << 23) : 0.f;
                    eref = emax;
                }
#pragma unroll
                for (int k = 0; k < NT; ++k) {
                    const int ee = ev[k] - eref + 127 + kFp8PShift;
                    pscale[k] = (ev[k] == 0 || ee <= 0) ? 0.f
                              : __uint_as_float((__float_as_uint(v_scale[k]) & 0x807fffffu) | ((uint32_t)ee << 23));
                }
            }
#pragma unroll
            for (int k = 0; k < NT; ++k) {
                const float e0 = ex2(sv[k][0] - m_new), e1 = ex2(sv[k][1] - m_new);
                const float e2 = ex2(sv[k][2] - m_new), e3 = ex2(sv[k][3] - m_new);
                esum += (e0 + e1) + (e2 + e3);
                if constexpr (kFp8) {
                    // fp16, 11 significant bits; the normaliser is the unrounded sum
                    p01[k] = pack_f16x2(e0 * pscale[k], e1 * pscale[k]);  // tokens 4q, 4q+1   (k slots 2q, 2q+1)
                    p23[k] = pack_f16x2(e2 * pscale[k], e3 * pscale[k]);  // tokens 4q+2, 4q+3 (k slots 2q+8, 2q+9)
                } else {
                    p01[k] = pack_bf16x2(e0, e1);
                    p23[k] = pack_bf16x2(e2, e3);
                    rsum += (bf16lo_to_f32(p01[k]) + bf16hi_to_f32(p01[k])) + (bf16lo_to_f32(p23[k]) + bf16hi_to_f32(p23[k]));
                }
            }
            lx_run = lx_run * alpha + esum;
            if constexpr (kFp8) l_run = lx_run;
            else l_run = l_run * alpha + rsum;
            if (__any_sync(kFull, alpha != 1.f) || beta != 1.f) {  // beta is warp-uniform
                // acc columns are heads 2*qlane, 2*qlane+1: fetch their alphas from those quads
                const float a_lo = __shfl_sync(kFull, alpha, (2 * qlane) << 2) * beta;
                const float a_hi = __shfl_sync(kFull, alpha, (2 * qlane + 1) << 2) * beta;
#pragma unroll
                for (int mt = 0; mt < C::kKSteps; ++mt) {
                    acc[mt][0] *= a_lo;
                    acc[mt][1] *= a_hi;
                    acc[mt][2] *= a_lo;
                    acc[mt][3] *= a_hi;
                }
            }

            // S5: O^T[16 d x 8 heads] += V^T[16 d x 16 tok] * P^T[16 tok x 8 heads]
            if constexpr (kFp8) {
                // ldmatrix.m16n16.trans.b8 hands each lane, per 16-token x 16-d byte block, the tokens 4q .. 4q+3 of
                // columns d = quad and quad + 8: the two byte pairs of a register widen (exactly) to the fp16 pairs
                // {a0 | a2} (row quad) and {a1 | a3} (row quad + 8) of the A fragment of m-tile mt -- the same
                // accumulator layout as the bf16 path, no byte shuffling.  One x2 load covers two m-tiles.
                const int lrow = lane & 15, lmat = lane >> 4;
#pragma unroll
                for (int k = 0; k < NT; ++k) {
#pragma unroll
                    for (int mp = 0; mp < C::kKSteps / 2; ++mp) {
                        const uint32_t chunk = (uint32_t)(2 * mp + lmat);
                        const uint32_t a = D == 128 ? v_base[k] + lrow * 128 + ((chunk ^ (uint32_t)(lrow & 7)) << 4)
                                                    : v_base[k] + lrow * 64 + (chunk << 4);
                        uint32_t r[4];
                        ldmatrix_b8_x2_trans(r, a);
                        mma_f16_16816(acc[2 * mp], e4m3x2_lo_to_f16x2(r[0]), e4m3x2_lo_to_f16x2(r[1]),
                                      e4m3x2_hi_to_f16x2(r[0]), e4m3x2_hi_to_f16x2(r[1]), p01[k], p23[k]);
                        mma_f16_16816(acc[2 * mp + 1], e4m3x2_lo_to_f16x2(r[2]), e4m3x2_lo_to_f16x2(r[3]),
                                      e4m3x2_hi_to_f16x2(r[2]), e4m3x2_hi_to_f16x2(r[3]), p01[k], p23[k]);
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < NT; ++k) {
#pragma unroll
                    for (int mt = 0; mt < C::kKSteps; ++mt) {
                        uint32_t vf[4];
                        const uint32_t chunk = ((2 * mt) & 7) | ld_half;
                        ldmatrix_x4_trans(vf, v_base[k] + (mt >> 2) * 2048 + ld_row_off + ((chunk ^ ld_xor) << 4));
                        mma_bf16_16816(acc[mt], vf[0], vf[1], vf[2], vf[3], p01[k], p23[k]);
                    }
                }
            }

            __syncwarp();
#pragma unroll
            for (int k = 0; k < NT; ++k) {
                if (lane == 0) mbar_arrive(empty0 + 8 * stg[k]);
                stage += kConsumerWarps;
                if (stage >= C::kStages) {
                    stage -= C::kStages;
                    phase ^= 1u;
                }
            }
            t += NT * kConsumerWarps;
        };
        if constexpr (C::kTilesPerPass == 2) {
            while (t + kConsumerWarps < n + cnt && !(kEarly && aborted)) tiles_pass(std::integral_constant<int, 2>{});
        }
        while (t < n + cnt && !(kEarly && aborted)) tiles_pass(std::integral_constant<int, 1>{});
        if (kEarly && early_pending) need_verdict();  // S6 stores to global memory
        if (kEarly && aborted) break;

        // S6: merge the consumer warps' states (warp-index order) and write the row or a partial.
        // Scratch layout per warp: acc as [head][D + 4] (the +4 pad makes both the fragment
        // scatter below and the float4 row reads after the barrier bank-conflict free), then m, l, lx.
        COMEM_STAMP(4);
        l_run += __shfl_xor_sync(kFull, l_run, 1);
        l_run += __shfl_xor_sync(kFull, l_run, 2);
        lx_run += __shfl_xor_sync(kFull, lx_run, 1);
        lx_run += __shfl_xor_sync(kFull, lx_run, 2);
        if constexpr (kFp8) {  // back to plain units: acc *= 2^(eref - 127 - kFp8PShift) (exact, unless it leaves the fp32 range)
            const int sh = eref - kFp8PShift;
            const float unit = sh <= 0 ? 0.f : __uint_as_float((uint32_t)(sh < 254 ? sh : 254) << 23);
#pragma unroll
            for (int mt = 0; mt < C::kKSteps; ++mt) {
                acc[mt][0] *= unit; acc[mt][1] *= unit; acc[mt][2] *= unit; acc[mt][3] *= unit;
            }
        }
        {
            float *lo = my_scratch + (2 * qlane) * C::kRowPitch + quad;
            float *hi = lo + C::kRowPitch;
#pragma unroll
            for (int mt = 0; mt < C::kKSteps; ++mt) {
                lo[16 * mt] = acc[mt][0];
                hi[16 * mt] = acc[mt][1];
                lo[16 * mt + 8] = acc[mt][2];
                hi[16 * mt + 8] = acc[mt][3];
            }
        }
        if (qlane == 0) {
            my_scratch[C::kStateOff + quad] = m_run;
            my_scratch[C::kStateOff + kMaxGroup + quad] = l_run;
            my_scratch[C::kStateOff + 2 * kMaxGroup + quad] = lx_run;
        }
        named_bar_sync(1, kConsumerThreads);
        if (warp < p.group) {  // warp w merges head w; lane -> one float4 of the row
            const int head = warp;
            float ww[kConsumerWarps], M = -INFINITY;
#pragma unroll
            for (int w = 0; w < kConsumerWarps; ++w) {
                ww[w] = scratch[w * C::kScratchFloatsPerWarp + C::kStateOff + head];
                M = fmaxf(M, ww[w]);
            }
            float den = 0.f, den_x = 0.f;
#pragma unroll
            for (int w = 0; w < kConsumerWarps; ++w) {
                ww[w] = ex2(ww[w] - M);  // a warp that saw no tile has m = -inf -> weight 0
                den += ww[w] * scratch[w * C::kScratchFloatsPerWarp + C::kStateOff + kMaxGroup + head];
                den_x += ww[w] * scratch[w * C::kScratchFloatsPerWarp + C::kStateOff + 2 * kMaxGroup + head];
            }
            const int64_t row = (int64_t)sp.b * p.num_q_heads + head0 + head;
            const int64_t rec = (int64_t)(x == c0 ? 0 : 1) * p.part_cap + cta;  // [kind][cta]
            if (lane < D / 4) {
                float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int w = 0; w < kConsumerWarps; ++w) {
                    const float4 a = *reinterpret_cast<const float4 *>(
                        scratch + w * C::kScratchFloatsPerWarp + head * C::kRowPitch + 4 * lane);
                    num.x += ww[w] * a.x; num.y += ww[w] * a.y; num.z += ww[w] * a.z; num.w += ww[w] * a.w;
                }
                if (whole_segment) {
                    const float inv = 1.f / den;
                    uint2 packed;
                    packed.x = pack_bf16x2(num.x * inv, num.y * inv);
                    packed.y = pack_bf16x2(num.z * inv, num.w * inv);
                    *reinterpret_cast<uint2 *>(p.out + row * D + 4 * lane) = packed;
                } else {
                    *reinterpret_cast<float4 *>(p.part_acc + rec * (kMaxGroup * D) + head * D + 4 * lane) = num;
                }
            }
            if (whole_segment) {
                if (p.lse_out && lane == 0) p.lse_out[row] = (M + log2f(den_x)) * 0.69314718055994530942f;
            } else if (lane < 2) {  // the head's state sector, written whole: {m, l, lx, 0} {0, 0, 0, 0}
                *reinterpret_cast<float4 *>(p.part_state + rec * kStateFloats + 8 * head + 4 * lane) =
                    lane == 0 ? make_float4(M, den, den_x, 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
        bool early_ticket = false;
        if (!whole_segment && p.fuse_combine) {
            // S7.  A cut segment that is not the CTA's last one (i.e. its first, with tiles of other
            // segments still to stream) must not stall the stream for the fence / ticket / merge round
            // trips (~3 us): thread 0 alone takes its ticket after the barrier below while the other
            // warps go on with the next segment; in mid-stream this CTA is practically never the last
            // arriver, and if it is, the merge waits until the CTA's end.
            if (x + cnt < c1) early_ticket = true;
            else {
                publish_and_merge(pending_first, true, x == c0 ? 0 : 1);
                pending_first = false;
            }
        }
        named_bar_sync(1, kConsumerThreads);
        if (early_ticket) {
            pending_first = true;
            if (threadIdx.x == 0) {
                int *ctr = p.seg_counters + s_seg[0][4];
                fence_acq_rel_gpu();  // after the barrier: covers every consumer's partial stores
                const int last0 = atomicAdd(ctr, 1) == s_seg[0][3] - 1;
                if (last0) *ctr = 0;
                s_seg[0][0] = last0;
            }
        }
        COMEM_STAMP(7);

        x += cnt;
        n += cnt;
    }
    if (pending_first && !(kEarly && aborted)) publish_and_merge(true, false, 0);  // the CTA's last segment was a whole one
    if (kEarly && aborted) {
        // every tile the producers issued before the verdict must have landed before the barriers are re-initialised:
        // this warp's share of them that it has not consumed
        for (int tt = t; tt < xp; tt += kConsumerWarps)
            mbar_wait(full0 + 8 * (tt & (C::kStages - 1)), (uint32_t)(tt / C::kStages) & 1u);
    }
    } while (attempt_end());
    }  // consumers
}

template <int D, bool kFp8, bool kEarly>
cudaError_t configure_once()
{
    static PerDeviceOnce once;
    return set_max_smem_once(decode_split_kernel<D, kFp8, kEarly>, (int)smem_bytes_for<D, kFp8>(kMaxBatch), once);
}

}  // namespace

size_t split_smem_bytes(int head_dim, int batch)
{
    return head_dim == 128 ? smem_bytes_for<128, false>(batch) : smem_bytes_for<64, false>(batch);
}

cudaError_t split_default_grid(int head_dim, int *grid_ctas)
{
    // one CTA per SM whatever the variant: each takes most of the SM's shared memory
    (void)head_dim;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    *grid_ctas = sms;
    return cudaSuccess;
}

template <int D, bool kFp8, bool kEarly>
static cudaError_t launch_instance(const CUtensorMap &tm_k, const CUtensorMap &tm_v, const CUtensorMap &tm_kh,
                                   const CUtensorMap &tm_vh, const DecodeParams &p, cudaLaunchConfig_t &cfg)
{
    const cudaError_t e = configure_once<D, kFp8, kEarly>();
    if (e != cudaSuccess) return e;
    cfg.blockDim = dim3(Cfg<D, kFp8>::kThreads);
    cfg.dynamicSmemBytes = smem_bytes_for<D, kFp8>(p.batch, p.fuse_combine != 0);
    return cudaLaunchKernelEx(&cfg, decode_split_kernel<D, kFp8, kEarly>, tm_k, tm_v, tm_kh, tm_vh, p);
}
template <int D, bool kFp8>
static cudaError_t launch_variant(const CUtensorMap &tm_k, const CUtensorMap &tm_v, const CUtensorMap &tm_kh,
                                  const CUtensorMap &tm_vh, const DecodeParams &p, cudaLaunchConfig_t &cfg)
{
    // the early-mode instance only where the mode can act (the flag is set and no sliding window)
    if (p.kv_immutable != 0 && p.window <= 0) return launch_instance<D, kFp8, true>(tm_k, tm_v, tm_kh, tm_vh, p, cfg);
    return launch_instance<D, kFp8, false>(tm_k, tm_v, tm_kh, tm_vh, p, cfg);
}

cudaError_t launch_decode_split(const CUtensorMap &tm_k, const CUtensorMap &tm_v, const DecodeParams &p,
                                int head_dim, cudaStream_t stream, bool kv_fp8, const CUtensorMap *tm_k_host,
                                const CUtensorMap *tm_v_host)
{
    // without a host tier the two extra descriptors are never used: pass the device ones
    const CUtensorMap &tm_kh = tm_k_host ? *tm_k_host : tm_k, &tm_vh = tm_v_host ? *tm_v_host : tm_v;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.grid_ctas);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p.no_pdl ? 0 : 1;
    if (kv_fp8)
        return head_dim == 128 ? launch_variant<128, true>(tm_k, tm_v, tm_kh, tm_vh, p, cfg)
                               : launch_variant<64, true>(tm_k, tm_v, tm_kh, tm_vh, p, cfg);
    if (head_dim == 128) return launch_variant<128, false>(tm_k, tm_v, tm_kh, tm_vh, p, cfg);
    return launch_variant<64, false>(tm_k, tm_v, tm_kh, tm_vh, p, cfg);
}

}  // namespace comem
