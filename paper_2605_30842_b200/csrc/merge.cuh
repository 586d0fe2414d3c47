// merge.cuh — S7, the log-sum-exp merge of one cut segment's split partials.
// Shared by K1 (fused: the last CTA to arrive on a segment runs it) and K2 (stand-alone combine).
#pragma once
#include "decode_params.cuh"
#include "ptx.cuh"
#include "schedule.cuh"

namespace comem {

constexpr unsigned kFullMask = 0xffffffffu;

// LSE merge of the `nsplit` partials of one cut segment by up to 8 warps of one CTA.  Warp w
// merges query head w of the group; lane -> one float4 of the head's D outputs.
//
// This code runs once per cut segment, at the very tail of the kernel, so two things matter more
// than arithmetic: (1) round trips to L2 -- all record loads of a round are put in flight together,
// the per-record scalars (m, l, lx) by lane = record into registers, the accumulator rows with
// cp.async (16 B per lane per record, L2-only) into a shared-memory staging area where every lane
// later reads back exactly the bytes it fetched; (2) code size -- the loops stay rolled, because
// fetching a few KiB of cold unrolled SASS costs more than the merge itself.
// Records are summed in split-index (= CTA-index) order with a running max; the arithmetic order
// is a function of the schedule only, never of which CTA runs the merge, so the row is
// bit-identical from run to run.
template <int D>
struct MergeCfg {
    static constexpr int kRecords = (D == 128) ? 20 : 32;  // records staged per round (<= 32: one per lane)
    static constexpr int kRecordFloats = kMaxGroup * D;     // staged part of a record: acc[8][D]
    static constexpr int kStageBytes = kRecords * kRecordFloats * 4;
};

template <int D>
__device__ __forceinline__ void merge_partials(const DecodeParams &p, int warp, int lane, int first_slot,
                                               int i_first, int nsplit, int64_t row0, float *stage)
{
    using MC = MergeCfg<D>;
    const int head = warp;
    if (head >= p.group) return;  // warp-uniform
    constexpr int kRowF4 = D / 4;                 // float4 per accumulator row: 32 or 16
    const bool active = lane < kRowF4;            // D = 64: lanes 16..31 only help with the scalars
    const int f4 = lane & (kRowF4 - 1);
    const int stride = partial_stride_floats(D);
    auto record = [&](int sidx) {
        return p.partials + (int64_t)(sidx == 0 ? first_slot : 2 * (i_first + sidx)) * stride;
    };
    float *mine = stage + head * D + 4 * f4;      // + i * kRecordFloats for the round's record i
    const uint32_t mine_s = smem_u32(mine);
    float M = -INFINITY, den = 0.f, den_x = 0.f;
    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
    for (int s0 = 0; s0 < nsplit; s0 += MC::kRecords) {
        const int n = min(MC::kRecords, nsplit - s0);
        float m_l = -INFINITY, l_l = 0.f, lx_l = 0.f;
        if (lane < n) {
            const float *rec_l = record(s0 + lane) + kMaxGroup * D + head;
            m_l = __ldcg(rec_l);
            l_l = __ldcg(rec_l + kMaxGroup);
            lx_l = __ldcg(rec_l + 2 * kMaxGroup);
        }
        if (active) {
#pragma unroll 4
            for (int i = 0; i < n; ++i)
                cp_async_16(mine_s + i * (MC::kRecordFloats * 4), record(s0 + i) + head * D + 4 * f4);
        }
#ifdef COMEM_TRACE
        if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 8] = globaltimer_ns() + (unsigned long long)(m_l == 12345.f);
#endif
        cp_async_wait_all();
#ifdef COMEM_TRACE
        if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 9] = globaltimer_ns();
#endif
        float bm = m_l;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bm = fmaxf(bm, __shfl_xor_sync(kFullMask, bm, o));
        bm = fmaxf(bm, M);
        const float r = (M == -INFINITY) ? 0.f : ex2(M - bm);  // bm >= M
        M = bm;
        const float w_l = (m_l == -INFINITY) ? 0.f : ex2(m_l - bm);
        const float wl_l = w_l * l_l, wlx_l = w_l * lx_l;
        den *= r;
        den_x *= r;
        num.x *= r; num.y *= r; num.z *= r; num.w *= r;
#pragma unroll 4
        for (int i = 0; i < n; ++i) {
            const float w = __shfl_sync(kFullMask, w_l, i);
            den += __shfl_sync(kFullMask, wl_l, i);
            den_x += __shfl_sync(kFullMask, wlx_l, i);
            if (active) {
                const float4 a = *reinterpret_cast<const float4 *>(mine + i * MC::kRecordFloats);
                num.x += w * a.x; num.y += w * a.y; num.z += w * a.z; num.w += w * a.w;
            }
        }
    }
#ifdef COMEM_TRACE
    if (p.trace && threadIdx.x == 0) p.trace[blockIdx.x * 16 + 10] = globaltimer_ns() + (unsigned long long)(den == 12345.f);
#endif
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
