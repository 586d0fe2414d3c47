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
// This code runs once per cut segment, at the very tail of the kernel, where what costs is
// (1) round trips to L2 and the number of requests one SM's load/store path keeps in flight -- a
// round's accumulator rows (G*D fp32, contiguous at the head of each record) are therefore fetched
// by the TMA unit, one bulk copy per record, all in flight at once, into a shared-memory staging
// area, and the per-record scalars (m, l, lx) by lane = record into registers meanwhile;
// (2) code size -- the loops stay rolled: fetching KiBs of cold unrolled SASS costs more than the math.
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
    static constexpr int kRecords = (D == 128) ? 20 : 32;  // records staged per round (<= 32: one per lane)
    static constexpr int kRecordFloats = kMaxGroup * D;     // staged part of a record: acc[8][D]
    static constexpr int kStageBytes = kRecords * kRecordFloats * 4;
};

template <int D>
__device__ __forceinline__ void merge_partials(const DecodeParams &p, int warp, int lane, int first_slot,
                                               int i_first, int nsplit, int64_t row0, float *stage,
                                               uint32_t mbar, uint32_t &phase)
{
    using MC = MergeCfg<D>;
    const int head = warp;
    constexpr int kRowF4 = D / 4;                               // float4 per accumulator row: 32 or 16
    const bool active = head < p.group && lane < kRowF4;         // D = 64: lanes 16..31 only help with the scalars
    const int f4 = lane & (kRowF4 - 1);
    const int stride = partial_stride_floats(D);
    const uint32_t rows_bytes = (uint32_t)p.group * D * 4;
    auto record = [&](int sidx) {
        return p.partials + (int64_t)(sidx == 0 ? first_slot : 2 * (i_first + sidx)) * stride;
    };
    const float *mine = stage + (head & (kMaxGroup - 1)) * D + 4 * f4;  // + i * kRecordFloats for record i
    float M = -INFINITY, den = 0.f, den_x = 0.f;
    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
    for (int s0 = 0; s0 < nsplit; s0 += MC::kRecords) {
        const int n = min(MC::kRecords, nsplit - s0);
        if (s0 > 0) named_bar_sync(1, 32 * kMaxGroup);  // every warp is done reading the previous round
        if (warp == 0) {
            if (lane == 0) {
                fence_proxy_async_global();
                mbar_arrive_expect_tx(mbar, (uint32_t)n * rows_bytes);
            }
            __syncwarp();
            if (lane < n)
                bulk_load(smem_u32(stage + lane * MC::kRecordFloats), record(s0 + lane), rows_bytes, mbar);
        }
        float m_l = -INFINITY, l_l = 0.f, lx_l = 0.f;
        if (lane < n && head < p.group) {
            const float4 st = __ldcg(reinterpret_cast<const float4 *>(record(s0 + lane) + kMaxGroup * D + 8 * head));
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
        const float wl_l = w_l * l_l, wlx_l = w_l * lx_l;
        den *= r;
        den_x *= r;
        num.x *= r; num.y *= r; num.z *= r; num.w *= r;
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
