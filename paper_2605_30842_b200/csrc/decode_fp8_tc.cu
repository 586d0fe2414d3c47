// decode_fp8_tc.cu — K1t, the split kernel of the decode step for the FP8 (E4M3 + per-page scale) cache of reading R18
// with BOTH contractions on the 5th-generation tensor cores (tcgen05.mma kind::f8f6f4, accumulators in TMEM), selected
// by COMEM_LAUNCH_FP8_TENSOR (D = 128, no sliding window).  Same step as decode_split.cu's FP8 instance (SURVEY.md
// section 8(a) S1..S6 for the cache of 8(f).3; "KV-cache quantisation", L49, L61), same schedule
// (schedule.cuh), same partial records; the merge (S7) is always the dependent combine kernel (combine.cu).
//
// Why: the warp-level path widens every E4M3 byte to fp16 in the consumer warps (64 conversions + 24 HMMA per 4 KiB
// stage) and is bound by their issue slots once the board's power cap lowers the SM clock.  The tensor core reads
// E4M3 operands straight from the TMA-swizzled tiles; the warps are left with the softmax.
//
// Transposed form, per SUPER TILE of 128 tokens (eight 16-token tiles of one (sequence, kv head) segment):
//     S^T[128 tok x 16] = K[128 tok x 128 d] . Qs^T          4 x (M 128, N 16, K 32); K and Qs K-major, 128-byte swizzle
//     O^T[128 d  x 16] += V^T[128 d x 128 tok] . Ps^T        4 x (M 128, N 16, K 32); V is the MN-major A operand
// The N = 16 columns are the group's 8 query heads x {hi, lo}: kind::f8f6f4 wants both operands in 8 bits, so a row of q
// (bf16, 8 significant bits) is scaled by a power of two and split EXACTLY into two E4M3 rows, q * 2^e = hi + lo / 16
// (exact for elements above 2^-14 of the row's largest), and a row of P the same way (p * v_scale, 8 significant bits
// after the split: the precision of the bf16 P of R16); the two accumulator columns are added in fp32.
//
// Roles (448 threads, one CTA per SM):
//   warps 0..7   softmax: two groups of four warps (thread = token row = TMEM lane); group g takes the super tiles
//                U = g (mod 2) of the CTA and keeps its own running maximum, normaliser and O accumulator, so the two
//                groups never wait for each other; their states are merged at the end of the segment (S6);
//   warp  8      prepares Qs per portion and issues S^T = K Qs^T, blocking on one barrier (the stage has landed); eight
//                S buffers in TMEM, so that the ring's own hand-off covers their reuse;
//   warp  9      issues O^T += V^T Ps^T, blocking on one barrier (the group's P tile is written), and frees the stage;
//   warps 10..13 producers: block table + page scales 32 tiles at a time (two batches ahead), one TMA box per 16-token
//                tile of K and of V into a 6-stage ring of 32 KiB super tiles (192 KiB in flight per SM).
// The running maximum is LAZY: a tile whose scores do not exceed it (one barrier.red.or over the group) goes straight to
// p = 2^(s - m); only a tile that raises it (or brings a page with a larger v_scale exponent) pays the cross-warp
// reduction and the rescale of O in TMEM.
#include "decode_params.cuh"
#include "ptx.cuh"
#include "schedule.cuh"
#include "tcgen05.cuh"

namespace comem {

namespace {

constexpr int kTcSoftmaxWarps = 8;
constexpr int kTcGroupThreads = 128;
constexpr int kTcMmaWarp = 8;
constexpr int kTcProducerWarps = 4;
constexpr int kTcPvWarp = 9;
constexpr int kTcFirstProducer = 10;
constexpr int kTcThreads = 32 * (kTcSoftmaxWarps + 2 + kTcProducerWarps);
constexpr int kTcD = 128;
constexpr int kSubTiles = 8;                       // 16-token tiles per super tile
constexpr int kSubBytes = kTileTokens * kTcD;      // one K (or V) tile: 2 KiB
constexpr int kHalfBytes = kSubTiles * kSubBytes;  // K (or V) part of a stage: 16 KiB
constexpr int kTcStageBytes = 2 * kHalfBytes;
constexpr int kTcStages = 6;                       // (5: +1.3 %, 4: +6 % on C4 in a burst)
constexpr int kSBufs = 8;                          // S^T buffers in TMEM (16 columns each); >= kTcStages + 2, see the QK warp
constexpr int kQBufs = 8;                          // Qs buffers (portion seg % 8)
constexpr int kTmemCols = 256;                     // S: columns 0..127, O of group g: 128 + 16 g
constexpr int kOCol = 128;
constexpr int kPShift = 7;                         // p * f * 2^(ev - eref) * 2^7 < 256 <= E4M3's 448
constexpr unsigned kFullMask32 = 0xffffffffu;
static_assert(kSBufs == 8 && kQBufs == 8, "buffer parities below are written for eight");


// shared-memory carve-up behind the 1024-aligned ring
struct TcSmem {
    static constexpr int kP = kTcStages * kTcStageBytes;  // 2 x 2 KiB: Ps of group 0 / 1
    static constexpr int kQ = kP + 2 * 2048;              // 8 x 2 KiB: Qs of portion seg % 8
    static constexpr int kAcc = kQ + kQBufs * 2048;            // S6: [2 groups][8 heads][128] fp32
    static constexpr int kState = kAcc + 2 * 8 * 128 * 4; // S6: m [2 groups][8], then l [2 groups][4 warps][8]
    static constexpr int kRed = kState + (16 + 64) * 4;   // lazy max: [2 groups][4 warps][8 + 1 (+ pad)] fp32
    static constexpr int kQc = kRed + 2 * 4 * 12 * 4;     // [8 buffers][8]: scale_log2 * 2^-e of the q rows
    static constexpr int kScales = kQc + kQBufs * 8 * 4;       // [stages][8 tiles] {k_scale, v_scale}
    static constexpr int kBars = kScales + kTcStages * kSubTiles * 8;
    static constexpr int kNumBars = 2 * kTcStages + kSBufs + 2 + 2 + kQBufs;  // full, empty, s_full, p_full, pv_done, q_full
    static constexpr int kPrefix = kBars + kNumBars * 8;
};
__host__ __device__ constexpr size_t tc_smem_bytes(int batch) { return 1024 + TcSmem::kPrefix + ((size_t)batch + 1) * 4 + 16; }
constexpr int kTcMaxBatch = 1024;  // (the prefix table of a larger batch does not fit beside the 192 KiB ring)
static_assert(tc_smem_bytes(kTcMaxBatch) <= 227 * 1024, "shared memory");

__host__ __device__ constexpr uint32_t umma_idesc_e4m3(int m, int n, bool a_mn_major, bool b_mn_major)
{
    // kind::f8f6f4: [4,6) D format (1 = f32), [7,10) A format (0 = E4M3), [10,13) B format (0 = E4M3)
    return (1u << 4) | ((a_mn_major ? 1u : 0u) << 15) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) |
           ((uint32_t)(m >> 4) << 24);
}
__device__ __forceinline__ void umma_f8_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
// shared-memory descriptor of an MN-major operand WITHOUT swizzle: 16 bytes of the M / N index contiguous, 8 contraction
// rows at a 16-byte pitch (a 128-byte core matrix), further groups of 8 rows lbo_bytes apart (probe-checked)
__device__ __forceinline__ uint64_t umma_smem_desc_mn_plain(uint32_t smem_addr, uint32_t lbo_bytes)
{
    return (uint64_t)((smem_addr & 0x3ffffu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | (1ull << 46);
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
// OR of a predicate over the `threads` threads that meet at named barrier `id`
__device__ __forceinline__ bool named_bar_or(int id, int threads, bool pred)
{
    uint32_t out;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t"
        "setp.ne.b32 p, %3, 0;\n\t"
        "barrier.cta.red.or.pred q, %1, %2, p;\n\t"
        "selp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(out) : "r"(id), "r"(threads), "r"((uint32_t)pred) : "memory");
    return out != 0;
}
// two fp32 -> two E4M3 bytes (round to nearest even, saturating): byte 0 = lo, byte 1 = hi
__device__ __forceinline__ uint32_t f32x2_to_e4m3x2(float lo, float hi)
{
    uint16_t r;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
    return r;
}
// two E4M3 bytes -> their exact values as fp32
__device__ __forceinline__ float2 e4m3x2_to_f32x2(uint32_t v)
{
    uint32_t h;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h) : "h"((uint16_t)v));
    float2 f;
    asm("{\n\t.reg .b16 a, b;\n\tmov.b32 {a, b}, %2;\n\tcvt.f32.f16 %0, a;\n\tcvt.f32.f16 %1, b;\n\t}" : "=f"(f.x), "=f"(f.y) : "r"(h));
    return f;
}
// x (|x| < 448) = hi + lo / 16 with hi, lo E4M3: returns {hi bytes of (a, b)} and {lo bytes} as byte pairs
__device__ __forceinline__ void split_e4m3x2(float a, float b, uint32_t &hi, uint32_t &lo)
{
    hi = f32x2_to_e4m3x2(a, b);
    const float2 back = e4m3x2_to_f32x2(hi);
    lo = f32x2_to_e4m3x2((a - back.x) * 16.f, (b - back.y) * 16.f);
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v) { asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
__device__ __forceinline__ float ex2f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

struct Portion {
    int b, kvh, j, T;  // sequence, kv head, first 16-token tile of the portion within the sequence, tiles in the sequence
    int cnt;           // 16-token tiles of this CTA's portion of the segment
};
__device__ __forceinline__ Portion locate_portion(int64_t x, int64_t c1, const int *prefix, int batch, int hkv)
{
    int lo = 0, hi = batch;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)hkv * prefix[mid] <= x) lo = mid; else hi = mid;
    }
    Portion s;
    s.b = lo;
    s.T = prefix[lo + 1] - prefix[lo];
    const int rel = (int)(x - (int64_t)hkv * prefix[lo]);
    s.kvh = rel / s.T;
    s.j = rel - s.kvh * s.T;
    const int64_t rem = c1 - x;
    s.cnt = (int)(rem < (int64_t)(s.T - s.j) ? rem : (int64_t)(s.T - s.j));
    return s;
}

// Walks the CTA's super tiles in order: portion after portion, kSubTiles tiles at a time.  Every role runs its own.
struct Cursor {
    int64_t x, c1;   // first linear tile of the current portion, end of the CTA's range
    Portion sp;
    int nsup;        // super tiles of the current portion
    int ul;          // super tile within the portion
    int U;           // CTA-local super tile index
    int seg;         // CTA-local portion index
    bool done;
    __device__ __forceinline__ void start(int64_t c0, int64_t c1_, const int *prefix, int batch, int hkv)
    {
        x = c0; c1 = c1_; ul = 0; U = 0; seg = 0;
        done = c0 >= c1_;
        if (!done) {
            sp = locate_portion(x, c1, prefix, batch, hkv);
            nsup = (sp.cnt + kSubTiles - 1) / kSubTiles;
        }
    }
    __device__ __forceinline__ void next(const int *prefix, int batch, int hkv)
    {
        ++U;
        if (++ul < nsup) return;
        x += sp.cnt;
        ul = 0;
        ++seg;
        if (x >= c1) { done = true; return; }
        sp = locate_portion(x, c1, prefix, batch, hkv);
        nsup = (sp.cnt + kSubTiles - 1) / kSubTiles;
    }
    __device__ __forceinline__ int sub_tiles() const { const int r = sp.cnt - ul * kSubTiles; return r < kSubTiles ? r : kSubTiles; }
};

__global__ void __launch_bounds__(kTcThreads, 1)
decode_fp8_tc_kernel(const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v, const DecodeParams p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;  // 1024-aligned: the 128B-swizzle atom
    uint8_t *sm = smem_raw + (base - raw);
    float *s6_acc = reinterpret_cast<float *>(sm + TcSmem::kAcc);
    float *s6_m = reinterpret_cast<float *>(sm + TcSmem::kState);  // [2 groups][8]
    float *s6_l = s6_m + 16;                                        // [2 groups][4 warps][8]
    float *red = reinterpret_cast<float *>(sm + TcSmem::kRed);      // [2 groups][4 warps][12]
    float *qc = reinterpret_cast<float *>(sm + TcSmem::kQc);        // [4 buffers][8]
    int *prefix = reinterpret_cast<int *>(sm + TcSmem::kPrefix);
    const uint32_t scales0 = base + TcSmem::kScales;
    const uint32_t full0 = base + TcSmem::kBars;
    const uint32_t empty0 = full0 + 8 * kTcStages;
    const uint32_t sfull0 = empty0 + 8 * kTcStages;
    const uint32_t pfull0 = sfull0 + 8 * kSBufs;
    const uint32_t pvdone0 = pfull0 + 16;
    const uint32_t qfull0 = pvdone0 + 16;

    __shared__ int s_e[kAlignedMaxSegs + 1];
    __shared__ int s_aligned, s_valid;
    __shared__ uint32_t s_tmem;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kTcStages; ++s) {
            mbar_init(full0 + 8 * s, kTcProducerWarps);
            mbar_init(empty0 + 8 * s, 1);
        }
        for (int s = 0; s < kSBufs; ++s) {
            mbar_init(sfull0 + 8 * s, 1);
            mbar_init(qfull0 + 8 * s, 1);
        }
        for (int g = 0; g < 2; ++g) {
            mbar_init(pfull0 + 8 * g, 4);
            mbar_init(pvdone0 + 8 * g, 1);
        }
        fence_mbar_init();
    }
    if (warp == kTcFirstProducer && lane == 0) {
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
    }
    if (warp == kTcMmaWarp) tmem_alloc<kTmemCols>(smem_u32(&s_tmem));
    // (as in decode_split.cu: hints only before the wait; the schedule is computed speculatively and validated after it)
    {
        const int64_t gtid = (int64_t)blockIdx.x * kTcThreads + threadIdx.x;
        if (gtid < (((int64_t)p.batch * 4 + 127) >> 7))
            prefetch_l2(reinterpret_cast<const char *>(p.seq_lens) + (gtid << 7));
        if (gtid < (((int64_t)p.batch * p.max_pages * 4 + 127) >> 7))
            prefetch_l2(reinterpret_cast<const char *>(p.block_table) + (gtid << 7));
        if (gtid < (((int64_t)p.batch * p.num_q_heads * kTcD * 2 + 127) >> 7))
            prefetch_l2(reinterpret_cast<const char *>(p.q) + (gtid << 7));
    }
    // S1: the schedule of schedule.cuh, decided exactly as decode_split.cu decides it (the combine kernel recomputes it)
    int64_t total = 0, c0 = 0, c1 = 0;
    const int cta = blockIdx.x;
    // (COMEM_DEBUG_STALE_GUESS=1, a testing aid as in decode_split.cu: the first schedule is computed from lengths 16 tokens short)
    int guess_bias = p.debug_stale_guess ? kTileTokens : 0;
    auto guess_len = [&](int L) { return L > guess_bias ? L - guess_bias : L; };
    auto compute_schedule = [&]() {
        if (warp == 0) {
            const int per = (p.batch + 31) >> 5;
            const int b0 = lane * per;
            int sum = 0;
#pragma unroll 1
            for (int i = 0; i < per; ++i)
                if (b0 + i < p.batch) sum += tiles_of(guess_len(__ldcg(p.seq_lens + b0 + i)));
            int incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(kFullMask32, incl, o);
                if (lane >= o) incl += v;
            }
            int run = incl - sum;
#pragma unroll 1
            for (int i = 0; i < per; ++i)
                if (b0 + i < p.batch) {
                    prefix[b0 + i] = run;
                    run += tiles_of(guess_len(__ldcg(p.seq_lens + b0 + i)));
                }
            if (lane == 31) prefix[p.batch] = incl;
            __syncwarp();
            const int S = p.batch * p.num_kv_heads;
            const int64_t tot = (int64_t)p.num_kv_heads * prefix[p.batch];
            bool ok = S <= kAlignedMaxSegs && tot >= (int64_t)gridDim.x * kMinTilesPerCta;
            if (ok) {
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
                ok = __all_sync(kFullMask32, mine_ok);
            }
            if (lane == 0) s_aligned = ok ? 1 : 0;
        }
        __syncthreads();
        total = (int64_t)p.num_kv_heads * prefix[p.batch];
        c0 = c1 = 0;
        if (total == 0) return;
        if (s_aligned) {
            int lo = 0, hi = p.batch * p.num_kv_heads;  // s_e[lo] <= cta < s_e[hi]
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (s_e[mid] <= cta) lo = mid; else hi = mid;
            }
            const int b = lo / p.num_kv_heads, kvh = lo - b * p.num_kv_heads;
            const int T = prefix[b + 1] - prefix[b];
            const int64_t seg0 = (int64_t)p.num_kv_heads * prefix[b] + (int64_t)kvh * T;
            const int al_first = s_e[lo], al_count = s_e[lo + 1] - al_first;
            c0 = aligned_cta_begin(seg0, T, cta - al_first, al_count);
            c1 = aligned_cta_begin(seg0, T, cta - al_first + 1, al_count);
        } else {
            const int nc = sched_num_ctas(total, (int)gridDim.x);
            if (cta < nc) {
                c0 = cta_begin(cta, total, nc);
                c1 = cta_begin(cta + 1, total, nc);
            }
        }
    };
    compute_schedule();  // speculative
    guess_bias = 0;
    const int tiles_per_page_mask = (1 << p.page_tile_shift) - 1;
    // tensor coordinates of tile jj of (sequence, kv head) in page pid: {d, token row, -, kv head}, or {d, slot, kv head, page} (HND)
    auto tile_coords = [&](int pid, int jj, int kvh, int &t1, int &t2, int &t3) {
        const int slot0 = (jj & tiles_per_page_mask) << kTileShift;
        t1 = p.kv_hnd ? slot0 : pid * p.page_size + slot0;
        t2 = p.kv_hnd ? kvh : 0;
        t3 = p.kv_hnd ? pid : kvh;
    };
    if (warp == kTcFirstProducer && c0 < c1) {  // L2 hint for the CTA's first tiles while the previous grid drains
        const Portion sp = locate_portion(c0, c1, prefix, p.batch, p.num_kv_heads);
        if (lane < sp.cnt) {
            const int jj = sp.j + lane;
            int page = jj >> p.page_tile_shift;
            page = page < p.max_pages ? page : p.max_pages - 1;
            const int pid = __ldcg(p.block_table + (int64_t)sp.b * p.max_pages + page);
            int t1, t2, t3;
            tile_coords(pid, jj, sp.kvh, t1, t2, t3);
            tma_prefetch_tile_4d(&tm_k, 0, t1, t2, t3);
            tma_prefetch_tile_4d(&tm_v, 0, t1, t2, t3);
        }
    }
    pdl_wait_prior_grid();
    if (warp == 0) {  // validate the guess against the lengths as they are now
        bool same = true;
#pragma unroll 1
        for (int b = lane; b < p.batch; b += 32)
            same = same && tiles_of(__ldcg(p.seq_lens + b)) == prefix[b + 1] - prefix[b];
        same = __all_sync(kFullMask32, same);
        if (lane == 0) s_valid = same ? 1 : 0;
    }
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    if (!s_valid) {
        __syncthreads();
        compute_schedule();
    }
    pdl_launch_dependents();
    const uint32_t tmem = s_tmem;

    if (warp >= kTcFirstProducer) {
        // ------------------------------ S2: page-gather producers ---------------------------------------------------
        // Producer pw loads the tiles in slots pw and pw + 4 of every super tile and arrives once per super tile.
        const int pw = warp - kTcFirstProducer;
        const uint64_t stream_policy = l2_policy_evict_first();
        int64_t x = c0;
        int stage = 0;
        uint32_t phase = 0;
        while (x < c1) {
            const Portion sp = locate_portion(x, c1, prefix, p.batch, p.num_kv_heads);
            const int cnt = sp.cnt;
            const int32_t *bt = p.block_table + (int64_t)sp.b * p.max_pages;
            // per-tile metadata (page id, then the page's two scales) 32 tiles at a time, two batches ahead of the TMAs
            auto load_pid = [&](int b0) -> int {
                if (b0 + lane >= cnt) return 0;
                return __ldg(bt + ((sp.j + b0 + lane) >> p.page_tile_shift));
            };
            auto load_scales = [&](int b0, int pid, float &ks, float &vs) {
                ks = vs = 0.f;
                if (b0 + lane < cnt) {
                    ks = __ldg(p.k_scale + (int64_t)pid * p.num_kv_heads + sp.kvh);
                    vs = __ldg(p.v_scale + (int64_t)pid * p.num_kv_heads + sp.kvh);
                }
            };
            int pid = load_pid(0), pid_next = load_pid(32);
            float ks, vs;
            load_scales(0, pid, ks, vs);
            for (int b0 = 0; b0 < cnt; b0 += 32) {
                float ks_next, vs_next;
                load_scales(b0 + 32, pid_next, ks_next, vs_next);
                const int pid_next2 = load_pid(b0 + 64);
#pragma unroll 1
                for (int uu = 0; uu < 4 && b0 + kSubTiles * uu < cnt; ++uu) {
                    const int la = kSubTiles * uu + pw, lb = la + 4;
                    const int sa = b0 + la, sb = b0 + lb;  // tile indices within the portion
                    mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                    const int pid_a = __shfl_sync(kFullMask32, pid, la), pid_b = __shfl_sync(kFullMask32, pid, lb);
                    const float ks_a = __shfl_sync(kFullMask32, ks, la), ks_b = __shfl_sync(kFullMask32, ks, lb);
                    const float vs_a = __shfl_sync(kFullMask32, vs, la), vs_b = __shfl_sync(kFullMask32, vs, lb);
                    if (elect_one()) {
                        const bool has_a = sa < cnt, has_b = sb < cnt;
                        const uint32_t bar = full0 + 8 * stage;
                        const uint32_t dst = base + stage * kTcStageBytes;
                        const uint32_t sc = scales0 + stage * (kSubTiles * 8);
                        if (has_a) asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(sc + 8 * pw), "f"(ks_a), "f"(vs_a) : "memory");
                        if (has_b) asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(sc + 8 * (pw + 4)), "f"(ks_b), "f"(vs_b) : "memory");
                        if (has_a) mbar_arrive_expect_tx(bar, (has_b ? 4u : 2u) * kSubBytes);
                        else mbar_arrive(bar);
                        int t1, t2, t3;
                        if (has_a) {
                            tile_coords(pid_a, sp.j + sa, sp.kvh, t1, t2, t3);
                            tma_load_4d_hint(dst + pw * kSubBytes, &tm_k, bar, 0, t1, t2, t3, stream_policy);
                            tma_load_4d_hint(dst + kHalfBytes + pw * kSubBytes, &tm_v, bar, 0, t1, t2, t3, stream_policy);
                        }
                        if (has_b) {
                            tile_coords(pid_b, sp.j + sb, sp.kvh, t1, t2, t3);
                            tma_load_4d_hint(dst + (pw + 4) * kSubBytes, &tm_k, bar, 0, t1, t2, t3, stream_policy);
                            tma_load_4d_hint(dst + kHalfBytes + (pw + 4) * kSubBytes, &tm_v, bar, 0, t1, t2, t3, stream_policy);
                        }
                    }
                    __syncwarp();
                    if (++stage == kTcStages) {
                        stage = 0;
                        phase ^= 1u;
                    }
                }
                pid = pid_next;
                pid_next = pid_next2;
                ks = ks_next;
                vs = vs_next;
            }
            x += cnt;
        }
    } else if (warp == kTcMmaWarp) {
        // ------------------------------ Qs, and S^T = K Qs^T ----------------------------------------------------------
        Cursor qk;
        qk.start(c0, c1, prefix, p.batch, p.num_kv_heads);
        int qk_stage = 0, prepared = -1;
        uint32_t qk_phase = 0;
        constexpr uint32_t idesc_qk = umma_idesc_e4m3(128, 16, false, false);
        // Qs of a portion: rows g (hi) and 8 + g (lo) of a [16][128 B] K-major tile, q[g] * 2^e = hi + lo / 16 with the
        // row's largest element scaled into [128, 256); qc[g] = scale_log2 * 2^-e.  Buffer seg % 8 (see below).
        auto prepare_q = [&](const Portion &sp, int seg) {
            const int buf = seg & (kQBufs - 1);
            const uint32_t qb = base + TcSmem::kQ + buf * 2048;
            const __nv_bfloat16 *q0 = p.q + ((int64_t)sp.b * p.num_q_heads + sp.kvh * p.group) * kTcD;
#pragma unroll 1
            for (int g8 = 0; g8 < kMaxGroup; ++g8) {
                uint2 w = make_uint2(0u, 0u);
                if (g8 < p.group) w = __ldg(reinterpret_cast<const uint2 *>(q0 + g8 * kTcD) + lane);
                const float f0 = __uint_as_float(w.x << 16), f1 = __uint_as_float(w.x & 0xffff0000u);
                const float f2 = __uint_as_float(w.y << 16), f3 = __uint_as_float(w.y & 0xffff0000u);
                float mx = fmaxf(fmaxf(fabsf(f0), fabsf(f1)), fmaxf(fabsf(f2), fabsf(f3)));
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(kFullMask32, mx, o));
                const int ebits = (int)((__float_as_uint(mx) >> 23) & 0xffu);
                int se = 261 - ebits;  // biased exponent of the scale 2^e, e = 134 - ebits
                se = se > 254 ? 254 : se;
                if (!(mx > 0.f) || ebits == 255) se = 127;  // a zero row; Inf / NaN rows propagate as they are
                const float scale = __uint_as_float((uint32_t)se << 23);
                uint32_t hi01, lo01, hi23, lo23;
                split_e4m3x2(f0 * scale, f1 * scale, hi01, lo01);
                split_e4m3x2(f2 * scale, f3 * scale, hi23, lo23);
                const uint32_t a = qb + g8 * 128 + ((((uint32_t)(lane >> 2) ^ (uint32_t)g8) << 4) | ((uint32_t)(lane & 3) << 2));
                sts32(a, hi01 | (hi23 << 16));
                sts32(a + 1024, lo01 | (lo23 << 16));
                if (lane == 0) qc[buf * 8 + g8] = p.scale_log2 * __uint_as_float((uint32_t)(254 - se) << 23);
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(qfull0 + 8 * buf);
        };
        // This warp issues S^T = K Qs^T only and waits on ONE barrier (the stage has landed), so it can block on it.
        // Nothing else gates it: S buffer U % 8 is free again when QK(U + 8) can be issued, because that needs ring
        // stage (U + 2) % 6 refilled, i.e. PV(U + 2) complete, i.e. the softmax group of U past its tile U + 2 -- and Qs
        // buffer seg % 8 likewise (a portion is at least one super tile).
        while (!qk.done) {
            if (prepared != qk.seg) {
                prepare_q(qk.sp, qk.seg);
                prepared = qk.seg;
            }
            mbar_wait(full0 + 8 * qk_stage, qk_phase);
            tc_fence_after_sync();
            if (elect_one()) {
                const uint32_t ka = base + qk_stage * kTcStageBytes, qb = base + TcSmem::kQ + (qk.seg & (kQBufs - 1)) * 2048;
                const uint32_t d = tmem + 16 * (qk.U & (kSBufs - 1));
#pragma unroll
                for (int ks = 0; ks < 4; ++ks)
                    umma_f8_ss(d, umma_smem_desc(ka + 32 * ks, 0, 1024), umma_smem_desc(qb + 32 * ks, 0, 1024), idesc_qk, ks > 0);
                umma_commit(sfull0 + 8 * (qk.U & (kSBufs - 1)));
            }
            __syncwarp();
            if (++qk_stage == kTcStages) {
                qk_stage = 0;
                qk_phase ^= 1u;
            }
            qk.next(prefix, p.batch, p.num_kv_heads);
        }
    } else if (warp == kTcPvWarp) {
        // ------------------------------ O^T += V^T Ps^T: one barrier (the group's P tile is written), blocking ----------
        // (One warp issuing both contractions was the kernel's critical resource: it polled two barriers and always
        // found both ready -- 1 413 cycles per tile; the two issuers never wait for each other.)
        Cursor pv;
        pv.start(c0, c1, prefix, p.batch, p.num_kv_heads);
        int pv_stage = 0;
        constexpr uint32_t idesc_pv = umma_idesc_e4m3(128, 16, true, true);
        while (!pv.done) {
            const int g = pv.U & 1;
            mbar_wait(pfull0 + 8 * g, (uint32_t)(pv.U >> 1) & 1u);
            tc_fence_after_sync();
            if (elect_one()) {
                const uint32_t va = base + pv_stage * kTcStageBytes + kHalfBytes, pb = base + TcSmem::kP + g * 2048;
                const uint32_t d = tmem + kOCol + 16 * g;
#pragma unroll
                for (int ks = 0; ks < 4; ++ks)
                    umma_f8_ss(d, umma_smem_desc(va + 4096 * ks, 0, 1024), umma_smem_desc_mn_plain(pb + 512 * ks, 128), idesc_pv,
                               (pv.ul >= 2 || ks > 0) ? 1u : 0u);
                umma_commit(empty0 + 8 * pv_stage);  // (QK of this stage completed before its softmax started)
                umma_commit(pvdone0 + 8 * g);
            }
            __syncwarp();
            if (++pv_stage == kTcStages) pv_stage = 0;
            pv.next(prefix, p.batch, p.num_kv_heads);
        }
    } else {
        // ------------------------------ softmax warps: S4, P, S6 ----------------------------------------------------
        const int g = warp >> 2, wq = warp & 3;
        const int t = 32 * wq + lane;  // token row of the super tile == TMEM lane; in S6: d
        const uint32_t lane_off = (uint32_t)(32 * wq) << 16;
        const uint32_t pbase = base + TcSmem::kP + g * 2048;
        // Ps is the MN-major B operand of O^T += V^T Ps^T, unswizzled: token t's 16 bytes {hi of heads 0..7, lo of heads
        // 0..7} are contiguous, so a thread hands over its token with ONE 16-byte store
        const uint32_t prow = pbase + 16 * t;
        Cursor cur;
        cur.start(c0, c1, prefix, p.batch, p.num_kv_heads);
        int stage = 0;
        while (!cur.done) {
            const Portion sp = cur.sp;
            const int seg = cur.seg, buf = seg & (kQBufs - 1);
            const int64_t x0 = cur.x;
            mbar_wait(qfull0 + 8 * buf, (uint32_t)(seg >> 3) & 1u);
            float c[kMaxGroup];
#pragma unroll
            for (int g8 = 0; g8 < kMaxGroup; ++g8) c[g8] = qc[buf * 8 + g8];
            const int seq_len = __ldcg(p.seq_lens + sp.b);
            float m[kMaxGroup], l[kMaxGroup];
#pragma unroll
            for (int g8 = 0; g8 < kMaxGroup; ++g8) {
                m[g8] = -INFINITY;
                l[g8] = 0.f;
            }
            int eref = 0, last_U = 0;
            bool has_o = false;
            for (;;) {
                if ((cur.U & 1) == g) {
                    const int U = cur.U;
                    const int tok0 = (sp.j + cur.ul * kSubTiles) << kTileShift;
                    int live = cur.sub_tiles() << kTileShift;
                    live = live < seq_len - tok0 ? live : seq_len - tok0;
                    const int sb = U & (kSBufs - 1);
                    mbar_wait(sfull0 + 8 * sb, (uint32_t)(U >> 3) & 1u);
                    tc_fence_after_sync();
                    uint32_t r[16];
                    tmem_ld16(tmem + lane_off + 16 * sb, r);
                    tmem_wait_ld();
                    float2 sc;
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(sc.x), "=f"(sc.y) : "r"(scales0 + stage * (kSubTiles * 8) + (t >> 4) * 8));
                    const bool dead = t >= live;
                    float s[kMaxGroup];
#pragma unroll
                    for (int g8 = 0; g8 < kMaxGroup; ++g8) {
                        const float v = fmaf(__uint_as_float(r[8 + g8]), 0.0625f, __uint_as_float(r[g8])) * (sc.x * c[g8]);
                        s[g8] = dead ? -INFINITY : v;  // masked by index, never by arithmetic
                    }
                    if (live < kSubTiles * kTileTokens && dead) {
                        // rows that do not count (past seq_len, or tiles this portion does not have) may hold anything,
                        // NaN bytes included: zero the V row so that 0 * NaN cannot reach the accumulator
                        const uint32_t vrow = base + stage * kTcStageBytes + kHalfBytes + t * 128;
#pragma unroll
                        for (int i = 0; i < 8; ++i) asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(vrow + 16 * i), "r"(0u) : "memory");
                    }
                    int ev = dead ? 0 : (int)((__float_as_uint(sc.y) >> 23) & 0xffu);
                    bool exceed = ev > eref;
#pragma unroll
                    for (int g8 = 0; g8 < kMaxGroup; ++g8) exceed = exceed || s[g8] > m[g8];
                    const bool raise = named_bar_or(1 + g, kTcGroupThreads, exceed);
                    // the group's previous P tile has been consumed and its PV has landed in O
                    if (U >= 2) {
                        mbar_wait(pvdone0 + 8 * g, ((uint32_t)(U >> 1) & 1u) ^ 1u);
                        tc_fence_after_sync();
                    }
                    if (raise) {
                        // the tile raises the running maximum of some head (or brings a larger v_scale exponent): exact
                        // tile maxima over the group's 128 rows, then O (TMEM) and l are brought to the new units
                        float tm[kMaxGroup];
#pragma unroll
                        for (int g8 = 0; g8 < kMaxGroup; ++g8) {
                            float v = s[g8];
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(kFullMask32, v, o));
                            tm[g8] = v;
                        }
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) ev = max(ev, __shfl_xor_sync(kFullMask32, ev, o));
                        float *rd = red + (g * 4 + wq) * 12;
                        if (lane < kMaxGroup) {
                            float mine = tm[0];
#pragma unroll
                            for (int g8 = 1; g8 < kMaxGroup; ++g8) mine = lane == g8 ? tm[g8] : mine;
                            rd[lane] = mine;
                        }
                        if (lane == 8) rd[8] = __int_as_float(ev);
                        named_bar_sync(1 + g, kTcGroupThreads);
                        const float *ra = red + g * 4 * 12;
                        int en = eref;
#pragma unroll
                        for (int w = 0; w < 4; ++w) en = max(en, __float_as_int(ra[w * 12 + 8]));
                        const int sh = 127 + eref - en;
                        const float beta = sh > 0 ? __uint_as_float((uint32_t)sh << 23) : 0.f;
                        float alpha[kMaxGroup];
#pragma unroll
                        for (int g8 = 0; g8 < kMaxGroup; ++g8) {
                            const float tmax = fmaxf(fmaxf(ra[g8], ra[12 + g8]), fmaxf(ra[24 + g8], ra[36 + g8]));
                            const float mn = fmaxf(m[g8], tmax);
                            alpha[g8] = (mn == m[g8]) ? 1.f : ex2f(m[g8] - mn);
                            m[g8] = mn;
                            l[g8] *= alpha[g8];
                        }
                        eref = en;
                        if (has_o) {
                            uint32_t o[16];
                            tmem_ld16(tmem + lane_off + kOCol + 16 * g, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int cc = 0; cc < 16; ++cc) o[cc] = __float_as_uint(__uint_as_float(o[cc]) * (alpha[cc & 7] * beta));
                            tmem_st16(tmem + lane_off + kOCol + 16 * g, o);
                            tmem_wait_st();
                        }
                    }
                    // p = 2^(s - m); the page's v_scale = f * 2^(ev - 127) rides on p as f * 2^(ev - eref + kPShift) < 256
                    float pscale;
                    {
                        const uint32_t vb = __float_as_uint(sc.y);
                        const int evt = (int)((vb >> 23) & 0xffu);
                        const int ee = evt - eref + 127 + kPShift;
                        pscale = (dead || evt == 0 || ee <= 0) ? 0.f : __uint_as_float((vb & 0x807fffffu) | ((uint32_t)ee << 23));
                    }
                    uint32_t hi[kMaxGroup / 2], lo[kMaxGroup / 2];
#pragma unroll
                    for (int i = 0; i < kMaxGroup / 2; ++i) {
                        const float p0 = ex2f(s[2 * i] - m[2 * i]), p1 = ex2f(s[2 * i + 1] - m[2 * i + 1]);
                        l[2 * i] += p0;
                        l[2 * i + 1] += p1;
                        split_e4m3x2(p0 * pscale, p1 * pscale, hi[i], lo[i]);
                    }
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(prow), "r"(hi[0] | (hi[1] << 16)),
                                 "r"(hi[2] | (hi[3] << 16)), "r"(lo[0] | (lo[1] << 16)), "r"(lo[2] | (lo[3] << 16)) : "memory");
                    fence_proxy_async_smem();
                    tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(pfull0 + 8 * g);
                    has_o = true;
                    last_U = U;
                }
                const bool last = cur.ul + 1 == cur.nsup;
                cur.next(prefix, p.batch, p.num_kv_heads);
                if (++stage == kTcStages) stage = 0;
                if (last) break;
            }
            // S6: the two groups' states -> the output row (the CTA owned the whole segment) or a partial record
            if (has_o) {
                mbar_wait(pvdone0 + 8 * g, (uint32_t)(last_U >> 1) & 1u);
                tc_fence_after_sync();
                uint32_t o[16];
                tmem_ld16(tmem + lane_off + kOCol + 16 * g, o);
                tmem_wait_ld();
                const int sh = eref - kPShift;  // back to plain units: 2^(eref - 127 - kPShift)
                const float unit = sh <= 0 ? 0.f : __uint_as_float((uint32_t)(sh < 254 ? sh : 254) << 23);
#pragma unroll
                for (int g8 = 0; g8 < kMaxGroup; ++g8) {
                    s6_acc[(g * 8 + g8) * kTcD + t] = fmaf(__uint_as_float(o[8 + g8]), 0.0625f, __uint_as_float(o[g8])) * unit;
                    float v = l[g8];
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(kFullMask32, v, off);
                    if (lane == g8) s6_l[(g * 4 + wq) * 8 + g8] = v;
                    if (wq == 0 && lane == g8) s6_m[g * 8 + g8] = m[g8];
                }
                tc_fence_before_sync();
            } else if (wq == 0 && lane < kMaxGroup) {
                s6_m[g * 8 + lane] = -INFINITY;
            }
            named_bar_sync(3, 32 * kTcSoftmaxWarps);
            {
                const int d = threadIdx.x & 127, half = threadIdx.x >> 7;
                const bool whole_segment = sp.j == 0 && sp.cnt == sp.T;
                const int64_t rec = (int64_t)(x0 == c0 ? 0 : 1) * p.part_cap + cta;  // [kind][cta]
#pragma unroll 1
                for (int hh = 0; hh < 4; ++hh) {
                    const int head = 4 * half + hh;
                    if (head >= p.group) break;
                    const float m0 = s6_m[head], m1 = s6_m[8 + head];
                    const float M = fmaxf(m0, m1);
                    const float w0 = m0 == -INFINITY ? 0.f : ex2f(m0 - M), w1 = m1 == -INFINITY ? 0.f : ex2f(m1 - M);
                    float den = 0.f, num = 0.f;
                    if (w0 != 0.f) {
                        const float *lp = s6_l + head;
                        den += w0 * ((lp[0] + lp[8]) + (lp[16] + lp[24]));
                        num += w0 * s6_acc[head * kTcD + d];
                    }
                    if (w1 != 0.f) {
                        const float *lp = s6_l + 32 + head;
                        den += w1 * ((lp[0] + lp[8]) + (lp[16] + lp[24]));
                        num += w1 * s6_acc[(8 + head) * kTcD + d];
                    }
                    const int64_t row = (int64_t)sp.b * p.num_q_heads + sp.kvh * p.group + head;
                    if (whole_segment) {
                        p.out[row * kTcD + d] = __float2bfloat16_rn(num / den);
                        if (p.lse_out && d == 0) p.lse_out[row] = (M + log2f(den)) * 0.69314718055994530942f;
                    } else {
                        p.part_acc[rec * (kMaxGroup * kTcD) + head * kTcD + d] = num;
                        if (d < 2)  // the head's state sector, written whole: {m, l, lx, 0} {0, 0, 0, 0}
                            *reinterpret_cast<float4 *>(p.part_state + rec * kStateFloats + 8 * head + 4 * d) =
                                d == 0 ? make_float4(M, den, den, 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
            }
            named_bar_sync(3, 32 * kTcSoftmaxWarps);
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    if (warp == kTcMmaWarp) tmem_dealloc<kTmemCols>(tmem);
}

}  // namespace

bool fp8_tc_supported(const DecodeParams &p, int head_dim)
{
    return head_dim == kTcD && p.window <= 0 && p.batch <= kTcMaxBatch;
}

cudaError_t launch_decode_fp8_tc(const CUtensorMap &tm_k, const CUtensorMap &tm_v, const DecodeParams &p, cudaStream_t stream)
{
    static PerDeviceOnce once;
    cudaError_t e = set_max_smem_once(decode_fp8_tc_kernel, (int)tc_smem_bytes(kTcMaxBatch), once);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.grid_ctas);
    cfg.blockDim = dim3(kTcThreads);
    cfg.dynamicSmemBytes = tc_smem_bytes(p.batch);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p.no_pdl ? 0 : 1;
    return cudaLaunchKernelEx(&cfg, decode_fp8_tc_kernel, tm_k, tm_v, p);
}

}  // namespace comem
