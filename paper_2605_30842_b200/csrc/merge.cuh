// merge.cuh — S7, the log-sum-exp merge of one cut segment's split partials.
// Shared by K1 (fused: the last CTA to arrive on a segment runs it) and K2 (stand-alone combine).
#pragma once
#include "decode_params.cuh"
#include "ptx.cuh"
#include "schedule.cuh"

namespace comem {

constexpr unsigned kFullMask = 0xffffffffu;

// LSE merge of the `nsplit` partials of one cut segment by the 8 warps (256 threads) of one CTA;
// ALL of them must call it (it syncs them on named barrier 1).  Warp w merges query head w of the
// group; lane -> one float4 of the head's D outputs.
//
// This code runs once per cut segment, at the very tail of the kernel, where what costs is round
// trips to L2 and instruction issue, not arithmetic:
//   * the accumulator rows of a round's records are fetched by the TMA unit into a shared-memory
//     staging area -- thanks to the [kind][cta] record layout (schedule.cuh) with TWO bulk copies
//     (the first split's record, then the contiguous run of the others), all bytes in flight at once;
//   * the per-record state {m, l, lx} is loaded by lane = record (one 16-byte L2 load) meanwhile;
//   * the weights go through a small per-warp shared array, so the accumulate loop is nothing
//     but independent LDS + FFMA;
//   * the loops stay rolled (cold straight-line SASS costs more to fetch than the math).
// Records are summed in split-index (= CTA-index) order with a running max; the arithmetic order
// is a function of the schedule only, never of which CTA runs the merge, so the row is
// bit-identical from run to run.
//
// Memory ordering: the partials were written with generic-proxy stores by other CTAs, each followed
// by a gpu-scope fence and its ticket (K1), or by a finished grid (K2); the caller has observed the
// last ticket and fenced (acquire).  The bulk copies read through the async proxy, straight from
// L2 (the point of coherence); fence.proxy.async.global below orders them after that acquire.
template <int D>
struct MergeCfg {
    static constexpr int kRecords = (D == 128) ? 19 : 32;  // records staged per round (<= 32: one per lane)
    static constexpr int kRecordFloats = kMaxGroup * D;     // acc[8][D]
    static constexpr int kWeightFloats = 4 * 32;            // per warp: {w, w*l, w*lx, 0} of the round's records
    static constexpr int kStageBytes = (kRecords * kRecordFloats + kMaxGroup * kWeightFloats) * 4;
};

template <int D>
__device__ __forceinline__ void merge_partials(const DecodeParams &p, int warp, int lane, int first_kind,
                                               int i_first, int nsplit, int64_t row0, float *stage,
                                               uint32_t mbar, uint32_t &phase)
{
    using MC = MergeCfg<D>;
    constexpr int RF = MC::kRecordFloats;
    const int head = warp;
    constexpr int kRowF4 = D / 4;                               // float4 per accumulator row: 32 or 16
    const bool active = head < p.group && lane < kRowF4;         // D = 64: lanes 16..31 only help with the state
    const int f4 = lane & (kRowF4 - 1);
    // record index of split s in the [kind][cta] arrays
    auto rec = [&](int sidx) { return sidx == 0 ? (int64_t)first_kind * p.part_cap + i_first : (int64_t)(i_first + sidx); };
    const float *mine = stage + (head & (kMaxGroup - 1)) * D + 4 * f4;  // + i * RF for the round's record i
    float *wb = stage + MC::kRecords * RF + warp * MC::kWeightFloats;
    float M = -INFINITY, den = 0.f, den_x = 0.f;
    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
    for (int s0 = 0; s0 < nsplit; s0 += MC::kRecords) {
        const int n = min(MC::kRecords, nsplit - s0);
        if (s0 > 0) named_bar_sync(1, 32 * kMaxGroup);  // every warp is done reading the previous round
        if (warp == 0 && lane == 0) {
            fence_proxy_async_global();
            mbar_arrive_expect_tx(mbar, (uint32_t)n * RF * 4);
            int i0 = 0;
            if (s0 == 0) {
                bulk_load(smem_u32(stage), p.part_acc + rec(0) * RF, RF * 4, mbar);
                i0 = 1;
            }
            if (n > i0)
                bulk_load(smem_u32(stage + i0 * RF), p.part_acc + rec(s0 + i0) * RF, (uint32_t)(n - i0) * RF * 4, mbar);
        }
        float m_l = -INFINITY, l_l = 0.f, lx_l = 0.f;
        if (lane < n && head < p.group) {
            const float4 st = __ldcg(reinterpret_cast<const float4 *>(p.part_state + rec(s0 + lane) * kStateFloats + 8 * head));
            m_l = st.x;
            l_l = st.y;
            lx_l = st.z;
        }
        float bm = m_l;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bm = fmaxf(bm, __shfl_xor_sync(kFullMask, bm, o));
        bm = fmaxf(bm, M);
        const float r = (M == -INFINITY) ? 0.f : ex2(M - bm);  // bm >= M
        M = bm;
        const float w_l = (m_l == -INFINITY) ? 0.f : ex2(m_l - bm);
        reinterpret_cast<float4 *>(wb)[lane] = make_float4(w_l, w_l * l_l, w_l * lx_l, 0.f);
        den *= r;
        den_x *= r;
        num.x *= r; num.y *= r; num.z *= r; num.w *= r;
        __syncwarp();
#ifdef COMEM_TRACE
        if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 8] = globaltimer_ns() + (unsigned long long)(m_l == 12345.f);
#endif
        mbar_wait(mbar, phase);
        phase ^= 1u;
#ifdef COMEM_TRACE
        if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 9] = globaltimer_ns();
#endif
#pragma unroll 4
        for (int i = 0; i < n; ++i) {
            const float4 w = reinterpret_cast<const float4 *>(wb)[i];  // one broadcast read
            den += w.y;
            den_x += w.z;
            if (active) {
                const float4 a = *reinterpret_cast<const float4 *>(mine + i * RF);
                num.x += w.x * a.x; num.y += w.x * a.y; num.z += w.x * a.z; num.w += w.x * a.w;
            }
        }
        __syncwarp();  // wb is rewritten by the next round
    }
#ifdef COMEM_TRACE
    if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 10] = globaltimer_ns() + (unsigned long long)(den == 12345.f);
#endif
    if (head >= p.group) return;
    const float inv = 1.f / den;
    const int64_t row = row0 + head;
    if (active) {
        uint2 packed;
        packed.x = pack_bf16x2(num.x * inv, num.y * inv);
        packed.y = pack_bf16x2(num.z * inv, num.w * inv);
        *reinterpret_cast<uint2 *>(p.out + row * D + 4 * f4) = packed;
    }
    if (p.lse_out && lane == 0) p.lse_out[row] = (M + log2f(den_x)) * 0.69314718055994530942f;
}

}  // namespace comem
