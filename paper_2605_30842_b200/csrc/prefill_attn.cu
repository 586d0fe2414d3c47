// prefill_attn.cu — K4, causal prefill attention over the paged KV cache (PAPER.md
// Algorithm 1 lines 9-13, L149-156: "Prefill new tokens only {Cached}" / "Prefill full context {Uncached}";
// L57-59: prefill is the compute-bound stage; L122: a full uncached prefill follows every summary adoption;
// DESIGN.md reading R20).  Sequence b's last n_b = q_start[b+1] - q_start[b] cached tokens are the new ones;
// query i of its chunk sits at position pos = L_b - n_b + i and attends the keys t <= pos:
//     out[row, h, :] = sum_{t <= pos} softmax_t(scale * q[row, h, :] . k_t[kvh, :]) v_t[kvh, :]
//
// This is the one dense contraction of the path, so it runs on the 5th-generation tensor cores
// (tcgen05.mma, accumulators in tensor memory), FlashAttention-style:
//   * work item = (sequence b, kv head, PAIR of 128-row query tiles).  A tile's 128 rows are R = 128 / G
//     consecutive positions x the G query heads of the kv head's group (row = position * G + head), so that
//     a K/V tile is fetched once for the whole GQA group; the two tiles of a pair share one K/V stream
//     (256 rows per 64 KiB of K+V: the L2 -> shared-memory traffic per flop that one tile would need is
//     above what the L2 delivers);
//   * warp 8 = producer: the pair's two Q tiles by one TMA load each (4-D box {64 d, G heads, R positions,
//     D/64}), then per 128-token KV block sixteen 8-token K half tiles and eight 16-token V tiles straight from the
//     block table (128-byte swizzle; V through the decode kernel's tensor map) into two-stage K and V rings;
//   * warp 9 = MMA issuer (one lane): S_t = Q_t K^T as D/16 instructions M128 N128 K16 -- K is loaded in HALF tiles of
//     8 token rows (a second tensor map over the pool, box {64, 8, D/64, 1}), so the 16 eight-row groups of a block sit
//     at one pitch (the descriptor's stride-dimension offset) and the whole block is one N dimension in token order.
//     (A shared-memory x shared-memory MMA re-reads its 4 KiB A slice of Q per instruction: two N = 64 instructions per
//     k-step, as the 16-row tiles forced, were bound by shared-memory bandwidth, 958 -> 1 060 TFLOP/s.)  O_t += P_t V as
//     one instruction M128 N(D) K16 per 16-token tile with P read from tensor memory and V, token-major in shared memory
//     exactly as the TMA laid it, as an MN-major operand;
//   * warps 0-3 / 4-7 = softmax of tile 0 / 1, one thread per row (TMEM lane = row): tcgen05.ld the 128
//     scores, causal mask by index, running max with a lazy rescale of O (only when the max grew by more
//     than 2^8; the accumulator rescale is a TMEM read-modify-write by the row's own thread), exp2, P rounded
//     to bf16 and written over the first 64 columns of S, l = sum of the ROUNDED p (reading R16);
//   * epilogue: O / l -> bf16 rows (and lse) by the row's thread.
// TMEM (512 columns): S0 | S1 (128 fp32 columns each, P aliased on their first 64) | O0 | O1 (D columns each).
// Everything that decides an output bit is a function of the logical problem (positions, never page ids),
// and a row is computed by one thread in a fixed order: results are bit-identical under page permutation.
#include <cstdio>
#include <type_traits>
#include "decode_params.cuh"
#include "prefill_params.cuh"
#include "ptx.cuh"
#include "tcgen05.cuh"

namespace comem {

namespace {

constexpr unsigned kAll = 0xffffffffu;
constexpr int kBlockTokens = 128;   // keys per KV block
constexpr int kTilesPerBlock = 8;   // 16-token TMA tiles per block
constexpr float kRescaleThreshold = 8.f;  // log2 domain: p stays below 2^8

template <int D>
struct PfCfg {
    static constexpr int kTileBytes = 16 * D * 2;                     // one 16-token K (or V) tile
    static constexpr int kStageBytes = kTilesPerBlock * kTileBytes;   // one 128-token K (or V) block
    static constexpr int kQTileBytes = 128 * D * 2;
    static constexpr int kKStages = 2, kVStages = 2;
    // 2 softmax warpgroups + a third warpgroup holding the producer warp, the MMA warp and two idle warps (a whole
    // warpgroup, so that it can hand its registers to the softmax warpgroups with setmaxnreg)
    static constexpr int kThreads = 384;
    static constexpr int kSoftmaxRegs = 208, kOtherRegs = 80;  // the CTA's own pool: 8 x (208 - 168) <= 4 x (168 - 80)
    static constexpr int kNumBars = 1 + 2 * kKStages + 2 * kVStages + 2 + 2 + 1;
    static constexpr int kSmemBytes = 1024 + 2 * kQTileBytes + (kKStages + kVStages) * kStageBytes + 8 * kNumBars + 64;
    static constexpr int kOCol = 256;     // TMEM column of O0; O1 follows at + D
};

#ifdef COMEM_PF_SPIN_LIMIT
__device__ __forceinline__ void pf_wait(uint32_t bar, uint32_t parity)
{
    for (long long i = 0; !mbar_try_wait(bar, parity); ++i)
        if (i > (long long)COMEM_PF_SPIN_LIMIT) {
            printf("prefill: barrier %u parity %u timed out (cta %d thread %d)\n", bar, parity, blockIdx.x, threadIdx.x);
            __trap();
        }
}
#else
__device__ __forceinline__ void pf_wait(uint32_t bar, uint32_t parity) { mbar_wait(bar, parity); }
#endif

__device__ __forceinline__ void tma_load_4d(uint32_t dst_smem, const void *tmap, uint32_t bar, int c0, int c1, int c2, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst_smem), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

// score column (S = Q K^T as issued: see the header) -> token of the 128-token block
__host__ __device__ constexpr int col_token(int col) { return col; }  // (K is laid out in token order: see the producer)

template <int D, bool kLse>
// (compiled at 168 registers, the most twelve warps can be launched with; the softmax warps then grow to 232)
__global__ void __launch_bounds__(PfCfg<D>::kThreads, 1)
prefill_attn_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                    const __grid_constant__ CUtensorMap tm_v, const PrefillParams p)
{
    using C = PfCfg<D>;
    extern __shared__ uint8_t smem_raw[];
    __shared__ uint32_t s_tmem;
    __shared__ int s_item[8];  // b, kvh, i0, n_b, L_b, q_start[b], found

    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t q_smem = base;                                  // [2 tiles][D/64][128 rows][128 B]
    const uint32_t k_smem = q_smem + 2 * C::kQTileBytes;           // [stage][8 tiles][D/64][16 rows][128 B]
    const uint32_t v_smem = k_smem + C::kKStages * C::kStageBytes;
    const uint32_t bars = v_smem + C::kVStages * C::kStageBytes;
    const uint32_t q_full = bars;
    const uint32_t k_full = q_full + 8, k_empty = k_full + 8 * C::kKStages;
    const uint32_t v_full = k_empty + 8 * C::kKStages, v_empty = v_full + 8 * C::kVStages;
    const uint32_t s_full = v_empty + 8 * C::kVStages;  // [2 tiles]
    const uint32_t p_full = s_full + 16;                 // [2 tiles]
    const uint32_t o_full = p_full + 16;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int R = p.rows_per_tile, G = p.group;

    // (thread 0; `again`: a persistent CTA starts its next work item with every barrier back in phase 0)
    auto init_barriers = [&](bool again) {
        auto one = [&](uint32_t bar, uint32_t count) {
            if (again) mbar_inval(bar);
            mbar_init(bar, count);
        };
        one(q_full, 1);
        for (int s = 0; s < C::kKStages; ++s) { one(k_full + 8 * s, 1); one(k_empty + 8 * s, 1); }
        for (int s = 0; s < C::kVStages; ++s) { one(v_full + 8 * s, 1); one(v_empty + 8 * s, 1); }
        for (int t = 0; t < 2; ++t) { one(s_full + 8 * t, 1); one(p_full + 8 * t, 4); }
        one(o_full, 1);
        fence_mbar_init();
    };
    if (threadIdx.x == 0) init_barriers(false);
    if (warp == 8 && lane == 0) {
        tma_prefetch_desc(&tm_q);
        tma_prefetch_desc(&tm_k);
        tma_prefetch_desc(&tm_v);
    }
    pdl_wait_prior_grid();  // q, q_start, seq_lens and the cache may come from the kernels queued before this one

    // ---- which work item: items are ordered (sequence, kv head, pair of query tiles from the LAST pair down) ----
    // (the CTAs resident together then stream the same kv head's cache, which stays in L2, and the long items run first).
    // A CTA takes the items blockIdx.x, blockIdx.x + gridDim.x, ...: with the default grid (one CTA per item) that is
    // one item; with comem_launch_opts.grid_ctas the kernel is persistent on that many SMs (the memory model's prefill
    // beside the agent's decode steps, section 5c of DESIGN.md).  Warp 0 looks the item up and publishes it in s_item.
    auto find_item = [&](const long long idx) {
        const int P2 = 2 * R, hkv = p.num_kv_heads;
        long long before = 0;  // pairs of the sequences before this chunk of 32
        int found = 0;
        for (int b0 = 0; b0 < p.batch && !found; b0 += 32) {
            const int b = b0 + lane;
            int n = 0, qs = 0;
            if (b < p.batch) {
                qs = __ldcg(p.q_start + b);
                n = __ldcg(p.q_start + b + 1) - qs;
            }
            const int np = n > 0 ? (n + P2 - 1) / P2 : 0;
            int incl = np;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(kAll, incl, o);
                if (lane >= o) incl += v;
            }
            const long long lo = (before + incl - np) * hkv, hi = (before + incl) * hkv;
            const unsigned hit = __ballot_sync(kAll, np > 0 && idx >= lo && idx < hi);
            if (hit) {
                const int src = __ffs(hit) - 1;
                if (lane == src) {
                    const int rel = (int)(idx - lo);
                    const int kvh = rel / np;
                    const int pair = np - 1 - (rel - kvh * np);
                    s_item[0] = b;
                    s_item[1] = kvh;
                    s_item[2] = pair * P2;
                    s_item[3] = n;
                    s_item[4] = __ldcg(p.seq_lens + b);
                    s_item[5] = qs;
                }
                found = 1;
            }
            before += __shfl_sync(kAll, incl, 31);
        }
        if (lane == 0) s_item[6] = found;
    };
// the published item, read by every thread after barrier A of the item loop
#define COMEM_PF_ITEM()                                                                                              \
    const int b = s_item[0], kvh = s_item[1], i0 = s_item[2], n_b = s_item[3], L_b = s_item[4], qs = s_item[5];       \
    const int nv = min(2 * R, n_b - i0);            /* valid positions of the pair */                                 \
    const bool act1 = nv > R;                        /* does tile 1 hold any valid row? */                             \
    const int pos0 = L_b - n_b + i0;                 /* position of the pair's first query */                          \
    const int kv_need = pos0 + nv;                   /* keys 0 .. pos_hi are needed, pos_hi = pos0 + nv - 1 */          \
    const int ntiles = (kv_need + 15) >> 4;                                                                           \
    const int nblk = (ntiles + kTilesPerBlock - 1) / kTilesPerBlock;                                                  \
    (void)b; (void)kvh; (void)qs; (void)act1; (void)L_b

    if (warp == 9) tmem_alloc<512>(smem_u32(&s_tmem));
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = s_tmem;

    // Item loop, once per role group (the register split must dominate each group's code).  Per item: barrier A (the
    // item is published, the barriers are fresh), the roles, barrier B (everybody is done with the item).
    if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::kOtherRegs));
    for (bool first = true;; first = false) {
    __syncthreads();  // A
    if (first) pdl_launch_dependents();
    if (!s_item[6]) break;  // past the last item (the grid is an upper bound on the number of items)
    COMEM_PF_ITEM();
    if (nblk <= 0) { __syncthreads(); continue; }  // n_b > L_b: invalid input (documented as undefined); no hang
    if (warp == 8) {
        // ------------------------------ producer -------------------------------------------------
        if (elect_one()) {
            const uint32_t qbytes = (uint32_t)(64 * G * R * (D / 64) * 2);
            mbar_arrive_expect_tx(q_full, act1 ? 2 * qbytes : qbytes);
            tma_load_4d(q_smem, &tm_q, q_full, 0, kvh * G, qs + i0, 0);
            if (act1) tma_load_4d(q_smem + C::kQTileBytes, &tm_q, q_full, 0, kvh * G, qs + i0 + R, 0);
        }
        const int32_t *bt = p.block_table + (int64_t)b * p.max_pages;
        const int tpm = (1 << p.page_tile_shift) - 1;
        for (int j = 0; j < nblk; ++j) {
            const int nt = min(kTilesPerBlock, ntiles - kTilesPerBlock * j);
            const int tile = kTilesPerBlock * j + lane;
            int row = 0;  // TMA row coordinate of this lane's tile: page * page_size + first slot
            if (lane < nt) row = __ldg(bt + (tile >> p.page_tile_shift)) * p.page_size + ((tile & tpm) << 4);
            const int sk = j % C::kKStages, sv = j % C::kVStages;
            pf_wait(k_empty + 8 * sk, ((uint32_t)(j / C::kKStages) & 1u) ^ 1u);
            if (elect_one()) mbar_arrive_expect_tx(k_full + 8 * sk, (uint32_t)nt * C::kTileBytes);
            for (int i = 0; i < nt; ++i) {
                const int r = __shfl_sync(kAll, row, i);
                // K in half tiles of 8 token rows (tm_k's box), 2 KiB each: [D/64 chunks][8 rows][128 B], so that the block's
                // 8-row groups sit at one pitch and the MMA takes all 128 tokens as its N dimension, in token order
                if (elect_one()) {
                    tma_load_4d(k_smem + sk * C::kStageBytes + i * C::kTileBytes, &tm_k, k_full + 8 * sk, 0, r, 0, kvh);
                    tma_load_4d(k_smem + sk * C::kStageBytes + i * C::kTileBytes + C::kTileBytes / 2, &tm_k, k_full + 8 * sk, 0,
                                r + 8, 0, kvh);
                }
            }
            pf_wait(v_empty + 8 * sv, ((uint32_t)(j / C::kVStages) & 1u) ^ 1u);
            if (elect_one()) mbar_arrive_expect_tx(v_full + 8 * sv, (uint32_t)nt * C::kTileBytes);
            for (int i = 0; i < nt; ++i) {
                const int r = __shfl_sync(kAll, row, i);
                if (elect_one()) tma_load_4d(v_smem + sv * C::kStageBytes + i * C::kTileBytes, &tm_v, v_full + 8 * sv, 0, r, 0, kvh);
            }
        }
    } else if (warp == 9) {
        // ------------------------------ MMA issuer -----------------------------------------------
        constexpr uint32_t idesc_qk = umma_idesc_bf16(128, kBlockTokens, false, false);
        constexpr uint32_t idesc_pv = umma_idesc_bf16(128, D, false, true);
        const int ntile_act = act1 ? 2 : 1;
        // S_t (block j) = Q_t K_j^T
        auto issue_qk = [&](int t, int j) {
            const uint32_t qb = q_smem + t * C::kQTileBytes, kb = k_smem + (j % C::kKStages) * C::kStageBytes;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const uint32_t c = ks >> 2, kin = (ks & 3) * 32;
                const uint64_t a = umma_smem_desc(qb + c * 16384 + kin, 0, 1024);
                // B: 16 groups of 8 token rows, C::kTileBytes / 2 apart; chunk c of a group at + c * 1 KiB
                const uint64_t bk = umma_smem_desc(kb + c * 1024 + kin, 0, C::kTileBytes / 2);
                umma_ss(tmem + 128 * t, a, bk, idesc_qk, ks > 0);
            }
        };
        // O_t += P_t V_j over the block's nt loaded tiles
        auto issue_pv = [&](int t, int j, int nt) {
            const uint32_t vb = v_smem + (j % C::kVStages) * C::kStageBytes;
            for (int i = 0; i < nt; ++i) {
                const uint64_t bd = umma_smem_desc(vb + i * C::kTileBytes, 2048, 1024);
                umma_ts(tmem + C::kOCol + D * t, tmem + 128 * t + 8 * i, bd, idesc_pv, (j > 0 || i > 0) ? 1u : 0u);
            }
        };
        pf_wait(q_full, 0);
        pf_wait(k_full, 0);
        tc_fence_after_sync();
        if (elect_one()) {
            for (int t = 0; t < ntile_act; ++t) {
                issue_qk(t, 0);
                umma_commit(s_full + 8 * t);
            }
            umma_commit(k_empty);
        }
        __syncwarp();
        for (int j = 0; j < nblk; ++j) {
            const int nt = min(kTilesPerBlock, ntiles - kTilesPerBlock * j);
            const int sv = j % C::kVStages;
            const bool more = j + 1 < nblk;
            const int skn = (j + 1) % C::kKStages;
            pf_wait(v_full + 8 * sv, (uint32_t)(j / C::kVStages) & 1u);
            // rows of the last tile that lie past the end of the sequence may hold anything (NaN included) and
            // 0 * NaN is NaN: zero them before the tensor core reads the tile (their P column is exactly 0)
            if (j == nblk - 1 && (L_b & 15) != 0 && (L_b >> 4) < ntiles) {
                const uint32_t tb = v_smem + sv * C::kStageBytes + ((L_b >> 4) - kTilesPerBlock * j) * C::kTileBytes;
                const int dead0 = L_b & 15;
                for (int idx = lane; idx < (16 - dead0) * (D / 8); idx += 32) {
                    const int rr = dead0 + idx / (D / 8), ch = idx % (D / 8);
                    asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(tb + (ch >> 3) * 2048 + rr * 128 + ((ch & 7) << 4)), "r"(0u) : "memory");
                }
                fence_proxy_async_smem();
                __syncwarp();
            }
            if (more) pf_wait(k_full + 8 * skn, (uint32_t)((j + 1) / C::kKStages) & 1u);
            for (int t = 0; t < ntile_act; ++t) {
                pf_wait(p_full + 8 * t, (uint32_t)j & 1u);
                tc_fence_after_sync();
                if (elect_one()) {
                    issue_pv(t, j, nt);
                    if (t == ntile_act - 1) umma_commit(v_empty + 8 * sv);
                    if (more) {
                        issue_qk(t, j + 1);
                        umma_commit(s_full + 8 * t);
                        if (t == ntile_act - 1) umma_commit(k_empty + 8 * skn);
                    }
                }
                __syncwarp();
            }
        }
        if (elect_one()) umma_commit(o_full);
        __syncwarp();
    }
    tc_fence_before_sync();
    __syncthreads();  // B
    }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::kSoftmaxRegs));
        for (long long idx = blockIdx.x;; idx += gridDim.x) {
        if (warp == 0) find_item(idx);
        if (threadIdx.x == 0 && idx != (long long)blockIdx.x) init_barriers(true);
        __syncthreads();  // A
        if (idx == (long long)blockIdx.x) pdl_launch_dependents();
        if (!s_item[6]) break;
        COMEM_PF_ITEM();
        if (nblk <= 0) { __syncthreads(); continue; }
        tc_fence_after_sync();
        // ------------------------------ softmax + epilogue: one thread per row ---------------------
        const int t = warp >> 2;                       // tile of the pair
        const int r = 32 * (warp & 3) + lane;          // row of the tile == TMEM lane
        const uint32_t lane_addr = (uint32_t)(32 * (warp & 3)) << 16;
        const uint32_t s_addr = tmem + lane_addr + 128 * t;
        const uint32_t o_addr = tmem + lane_addr + C::kOCol + D * t;
        if (t == 0 || act1) {
            const int ri = r / G, rg = r - ri * G;       // position within the tile, head within the group
            const int pos = pos0 + t * R + ri;           // this row's query position (meaningless for dead rows)
            const bool live = r < R * G && t * R + ri < nv;
            const int pos_lo = pos0 + t * R;             // smallest position of the tile
            float m_used = -INFINITY, l_run = 0.f, lx_run = 0.f;
            for (int j = 0; j < nblk; ++j) {
                pf_wait(s_full + 8 * t, (uint32_t)j & 1u);
                tc_fence_after_sync();
                float s[128];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    uint32_t u[32];
                    tmem_ld32(s_addr + 32 * c, u);
#pragma unroll
                    for (int i = 0; i < 32; ++i) s[32 * c + i] = __uint_as_float(u[i]);
                }
                tmem_wait_ld();
                const bool masked = kBlockTokens * j + kBlockTokens - 1 > pos_lo;  // uniform over the tile
                const int pos_rel = pos - kBlockTokens * j;
                if (masked) {
#pragma unroll
                    for (int c = 0; c < 128; ++c)
                        if (col_token(c) > pos_rel) s[c] = -INFINITY;
                }
                // (eight independent chains, then a tree: one thread per row means the row's 128 scores are one
                // thread's instruction stream, and a single 127-deep fmax chain is 127 dependent issue slots)
                float mr8[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) mr8[i] = s[i];
#pragma unroll
                for (int c = 8; c < 128; ++c) mr8[c & 7] = fmaxf(mr8[c & 7], s[c]);
                const float mr = fmaxf(fmaxf(fmaxf(mr8[0], mr8[1]), fmaxf(mr8[2], mr8[3])),
                                       fmaxf(fmaxf(mr8[4], mr8[5]), fmaxf(mr8[6], mr8[7])));
                const float mx = (mr == -INFINITY) ? -INFINITY : mr * p.scale_log2;
                const bool grow = mx > m_used + kRescaleThreshold;  // also the first block (m_used = -inf)
                float factor = 1.f;
                if (grow) {
                    factor = ex2(m_used - mx);  // 0 on the first block
                    m_used = mx;
                    l_run *= factor;
                    lx_run *= factor;
                }
                if (j > 0 && __any_sync(kAll, grow)) {
                    // O_t is idle here: PV(t, j-1) completed before S_t(j) was signalled, PV(t, j) waits for p_full
#pragma unroll
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t o[32];
                        tmem_ld32(o_addr + 32 * c, o);
                        tmem_wait_ld();
#pragma unroll
                        for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * factor);
                        tmem_st32(o_addr + 32 * c, o);
                    }
                }
                // p = 2^(s * scale - m), rounded to bf16; P word i holds tokens 2i, 2i+1 of the block.  Two copies of the
                // loop, chosen once per block: only the blocks on the diagonal carry the per-element mask test (a
                // predicated-off FSEL still takes its issue slot, and this loop is what the tensor pipe waits for), and
                // the unrounded sum is kept only when the caller wants lse_out.
                const float neg_m = -m_used;
                auto exp_pass = [&](auto masked_tag) {
                    constexpr bool kMasked = decltype(masked_tag)::value;
                    float rs4[4] = {0.f, 0.f, 0.f, 0.f};  // independent partial sums (fixed order)
                    [[maybe_unused]] float xs4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint32_t pw[32];
#pragma unroll
                        for (int i = 0; i < 32; ++i) {
                            const int col = 2 * (32 * h + i);              // P word w = 32 h + i: tokens 2w, 2w + 1 of the block
                            float e0 = ex2(fmaf(s[col], p.scale_log2, neg_m));
                            float e1 = ex2(fmaf(s[col + 1], p.scale_log2, neg_m));
                            if constexpr (kMasked) {  // (s = -inf and scale = 0 would give NaN above: decide by index)
                                if (col_token(col) > pos_rel) e0 = 0.f;
                                if (col_token(col + 1) > pos_rel) e1 = 0.f;
                            }
                            pw[i] = pack_bf16x2(e0, e1);
                            rs4[i & 3] += bf16lo_to_f32(pw[i]) + bf16hi_to_f32(pw[i]);
                            if constexpr (kLse) xs4[i & 3] += e0 + e1;
                        }
                        tmem_st32(s_addr + 32 * h, pw);
                    }
                    l_run += (rs4[0] + rs4[1]) + (rs4[2] + rs4[3]);
                    if constexpr (kLse) lx_run += (xs4[0] + xs4[1]) + (xs4[2] + xs4[3]);
                };
                if (masked) exp_pass(std::true_type{});
                else exp_pass(std::false_type{});
                tmem_wait_st();
                tc_fence_before_sync();
                __syncwarp();   // one arrival per warp (four per tile) instead of 128 serialised ones on one barrier
                if (lane == 0) mbar_arrive(p_full + 8 * t);
            }
            // epilogue
            pf_wait(o_full, 0);
            tc_fence_after_sync();
            const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
            const int64_t grow_idx = (int64_t)qs + i0 + t * R + ri;
            __nv_bfloat16 *orow = p.out + (grow_idx * p.num_q_heads + kvh * G + rg) * D;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t o[32];
                tmem_ld32(o_addr + 32 * c, o);
                tmem_wait_ld();
                if (live) {
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        uint4 w;
                        w.x = pack_bf16x2(__uint_as_float(o[8 * v]) * inv, __uint_as_float(o[8 * v + 1]) * inv);
                        w.y = pack_bf16x2(__uint_as_float(o[8 * v + 2]) * inv, __uint_as_float(o[8 * v + 3]) * inv);
                        w.z = pack_bf16x2(__uint_as_float(o[8 * v + 4]) * inv, __uint_as_float(o[8 * v + 5]) * inv);
                        w.w = pack_bf16x2(__uint_as_float(o[8 * v + 6]) * inv, __uint_as_float(o[8 * v + 7]) * inv);
                        *reinterpret_cast<uint4 *>(orow + 32 * c + 8 * v) = w;
                    }
                }
            }
            if constexpr (kLse) {
                if (live && p.lse_out)
                    p.lse_out[grow_idx * p.num_q_heads + kvh * G + rg] = (m_used + log2f(lx_run)) * 0.69314718055994530942f;
            }
        }
        tc_fence_before_sync();
        __syncthreads();  // B
        }
    }
#undef COMEM_PF_ITEM
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 9) tmem_dealloc<512>(tmem);
}

template <int D, bool kLse>
cudaError_t configure_prefill()
{
    static PerDeviceOnce once;
    return set_max_smem_once(prefill_attn_kernel<D, kLse>, PfCfg<D>::kSmemBytes, once);
}

template <int D, bool kLse>
cudaError_t launch_prefill_inst(const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                                const PrefillParams &p, cudaLaunchConfig_t &cfg)
{
    const cudaError_t e = configure_prefill<D, kLse>();
    if (e != cudaSuccess) return e;
    cfg.blockDim = dim3(PfCfg<D>::kThreads);
    cfg.dynamicSmemBytes = PfCfg<D>::kSmemBytes;
    return cudaLaunchKernelEx(&cfg, prefill_attn_kernel<D, kLse>, tm_q, tm_k, tm_v, p);
}

// (the instance without lse_out skips the unrounded row sums: one FADD per score in the loop the tensor pipe waits for)
template <int D>
cudaError_t launch_prefill_variant(const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                                   const PrefillParams &p, cudaLaunchConfig_t &cfg)
{
    return p.lse_out ? launch_prefill_inst<D, true>(tm_q, tm_k, tm_v, p, cfg)
                     : launch_prefill_inst<D, false>(tm_q, tm_k, tm_v, p, cfg);
}

}  // namespace

cudaError_t launch_prefill_attn(const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                                const PrefillParams &p, int head_dim, int grid, cudaStream_t stream, bool pdl)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    if (head_dim == 128) return launch_prefill_variant<128>(tm_q, tm_k, tm_v, p, cfg);
    return launch_prefill_variant<64>(tm_q, tm_k, tm_v, p, cfg);
}

}  // namespace comem
