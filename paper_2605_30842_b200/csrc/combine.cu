// combine.cu — K2, the stand-alone log-sum-exp combine.
//
// One CTA per (sequence b, kv head) segment, one warp per query head of the group.  It recomputes
// the same schedule as the split kernel (schedule.cuh) to learn which CTAs cut this segment, then
// runs merge.cuh's merge_partials over their fp32 partials (acc, m, l, lx), in CTA-index order:
//     M = max_s m_s;  w_s = 2^(m_s - M);  out = (sum_s w_s acc_s) / (sum_s w_s l_s)
// (l sums the bf16-rounded p and normalises out; lx sums the unrounded p and only feeds lse_out).
// Segments owned by a single CTA were already written by the split kernel and are skipped;
// empty sequences (seq_len == 0) get +0.0 rows and lse = -inf here (reading R9).
// Visibility of the partials comes from the grid dependency (this kernel starts its reads after
// the split grid has completed and flushed), so K1 needs no fence or ticket in this mode.
#include "decode_params.cuh"
#include "merge.cuh"
#include "ptx.cuh"
#include "schedule.cuh"

namespace comem {

namespace {

constexpr int kCombineThreads = 32 * kMaxGroup;  // warp w <-> query head w of the group

template <int D>
__global__ void __launch_bounds__(kCombineThreads)
combine_kernel(const DecodeParams p)
{
    extern __shared__ __align__(128) float stage[];  // MergeCfg<D>::kStageBytes
    __shared__ int s_before[kMaxGroup], s_total[kMaxGroup];
    __shared__ int s_prefix[kAlignedMaxSegs + 1], s_e[kAlignedMaxSegs + 1], s_aligned;
    __shared__ __align__(8) uint64_t s_bar;
    const int b = blockIdx.x / p.num_kv_heads;
    const int kvh = blockIdx.x - b * p.num_kv_heads;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    if (tid == 0) {
        mbar_init(smem_u32(&s_bar), 1);
        fence_mbar_init();
    }
    pdl_wait_prior_grid();  // seq_lens / partials come from the kernels launched just before

    // tiles before sequence b, and in total (block reduction over seq_lens)
    {
        int before = 0, total = 0;
#pragma unroll 1
        for (int i = tid; i < p.batch; i += kCombineThreads) {
            const int ti = seq_tiles(__ldg(p.seq_lens + i), p.window, p.sinks);
            total += ti;
            if (i < b) before += ti;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            before += __shfl_xor_sync(kFullMask, before, o);
            total += __shfl_xor_sync(kFullMask, total, o);
        }
        if (lane == 0) { s_before[warp] = before; s_total[warp] = total; }
        // the segment-aligned variant of the schedule (schedule.cuh), decided exactly as K1 decides it
        if (tid == 0) {
            s_aligned = 0;
            if (p.batch * p.num_kv_heads <= kAlignedMaxSegs) {
                s_prefix[0] = 0;
                for (int i = 0; i < p.batch; ++i) s_prefix[i + 1] = s_prefix[i] + seq_tiles(__ldg(p.seq_lens + i), p.window, p.sinks);
                if (s_prefix[p.batch] > 0)
                    s_aligned = aligned_build(s_prefix, p.batch, p.num_kv_heads, p.grid_ctas, s_e) ? 1 : 0;
            }
        }
    }
    __syncthreads();
    pdl_launch_dependents();
    int before = 0, total_tiles = 0;
#pragma unroll
    for (int w = 0; w < kMaxGroup; ++w) { before += s_before[w]; total_tiles += s_total[w]; }

    const int T = seq_tiles(__ldg(p.seq_lens + b), p.window, p.sinks);
    const int64_t row0 = (int64_t)b * p.num_q_heads + kvh * p.group;
    if (T == 0) {
        for (int e = tid; e < p.group * D; e += kCombineThreads) p.out[row0 * D + e] = __float2bfloat16_rn(0.f);
        if (p.lse_out && tid < p.group) p.lse_out[row0 + tid] = -INFINITY;
        return;
    }
    if (s_aligned) {
        const int sidx = b * p.num_kv_heads + kvh;
        const int c = s_e[sidx + 1] - s_e[sidx];
        if (c <= 1) return;
        uint32_t ph = 0;
        merge_partials<D>(p, warp, lane, 0, s_e[sidx], c, row0, stage, smem_u32(&s_bar), ph);
        return;
    }
    const int64_t total = (int64_t)p.num_kv_heads * total_tiles;
    const int nc = sched_num_ctas(total, p.grid_ctas);
    const int64_t seg0 = (int64_t)p.num_kv_heads * before + (int64_t)kvh * T;
    const int64_t seg1 = seg0 + T;
    const int i_first = cta_of_tile(seg0, total, nc);
    const int i_last = cta_of_tile(seg1 - 1, total, nc);
    if (i_first == i_last) return;  // one CTA owned the whole segment and wrote the rows itself
    // the first split's record is CTA i_first's kind-1 record when the segment starts inside its range
    const int first_slot = cta_begin(i_first, total, nc) < seg0 ? 1 : 0;
    uint32_t phase = 0;
    merge_partials<D>(p, warp, lane, first_slot, i_first, i_last - i_first + 1, row0, stage, smem_u32(&s_bar), phase);
}

// K2s, the SMALL dependent combine (COMEM_LAUNCH_SPLIT_COMBINE): the same merge for a step of few long segments
// (batch * Hkv <= kAlignedMaxSegs), shaped to sit BESIDE the split kernel on the SMs it occupies and to cost one
// round trip to L2 once that grid has drained:
//   * one CTA of 128 threads per (segment, query head), a few KiB of shared memory, launched with programmatic
//     stream serialization right behind K1.  K1 triggers its dependents after its own griddepcontrol.wait, so these
//     CTAs become resident while K1 streams; they trigger THEIR dependents at once (the next step's K1 may take
//     every SM K1 frees), work out which CTAs cut their segment (seq_lens is final: K1's wait has passed), and
//     park in griddepcontrol.wait;
//   * when K1's grid has completed and flushed, lane -> one float4 of the head's row, warp w -> the records
//     w, w + 4, ... of the segment: all loads of up to 20 records are issued before the first is used.  The weights
//     are taken against the segment's global maximum (known before any accumulation), each warp sums its records in
//     index order and the four warp sums are added in warp order: a fixed order, a function of the schedule only.
// K1 then needs neither fence nor ticket, and no CTA of it finishes later than the others because it merged.
#ifndef COMEM_SMALL_THREADS
#define COMEM_SMALL_THREADS 128
#endif
constexpr int kSmallThreads = COMEM_SMALL_THREADS;
constexpr int kSmallStripes = kSmallThreads / 32;
constexpr int kSmallBatch = 5;  // records per warp in flight

template <int D>
__global__ void __launch_bounds__(kSmallThreads)
combine_small_kernel(const DecodeParams p)
{
    __shared__ int s_prefix[kAlignedMaxSegs + 1], s_e[kAlignedMaxSegs + 1];
    __shared__ int s_info[4];  // tiles of the segment, record kind of its first split, first CTA, number of splits
    __shared__ __align__(16) float s_num[kSmallStripes][D];
    __shared__ float s_den[kSmallStripes][2];
    const int seg = blockIdx.x / p.group, head = blockIdx.x - seg * p.group;
    const int b = seg / p.num_kv_heads, kvh = seg - b * p.num_kv_heads;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    pdl_launch_dependents();
    if (tid == 0) {
        s_prefix[0] = 0;
        for (int i = 0; i < p.batch; ++i) s_prefix[i + 1] = s_prefix[i] + seq_tiles(__ldcg(p.seq_lens + i), p.window, p.sinks);
        const int T = s_prefix[b + 1] - s_prefix[b];
        int kind = 0, i_first = 0, nsplit = 0;
        if (T > 0) {
            if (aligned_build(s_prefix, p.batch, p.num_kv_heads, p.grid_ctas, s_e)) {
                i_first = s_e[seg];
                nsplit = s_e[seg + 1] - s_e[seg];
            } else {
                const int64_t total = (int64_t)p.num_kv_heads * s_prefix[p.batch];
                const int nc = sched_num_ctas(total, p.grid_ctas);
                const int64_t seg0 = (int64_t)p.num_kv_heads * s_prefix[b] + (int64_t)kvh * T;
                i_first = cta_of_tile(seg0, total, nc);
                nsplit = cta_of_tile(seg0 + T - 1, total, nc) - i_first + 1;
                kind = cta_begin(i_first, total, nc) < seg0 ? 1 : 0;
            }
        }
        s_info[0] = T; s_info[1] = kind; s_info[2] = i_first; s_info[3] = nsplit;
    }
    __syncthreads();
    const int T = s_info[0], kind = s_info[1], i_first = s_info[2], nsplit = s_info[3];
#ifdef COMEM_TRACE
    if (p.trace && tid == 0) p.trace[(1024 + blockIdx.x) * 16 + 0] = globaltimer_ns();
#endif
    pdl_wait_prior_grid();
#ifdef COMEM_TRACE
    if (p.trace && tid == 0) p.trace[(1024 + blockIdx.x) * 16 + 1] = globaltimer_ns();
#endif

    const int64_t row = (int64_t)b * p.num_q_heads + kvh * p.group + head;
    if (T == 0) {  // S8 (reading R9)
        for (int e = tid; e < D; e += kSmallThreads) p.out[row * D + e] = __float2bfloat16_rn(0.f);
        if (p.lse_out && tid == 0) p.lse_out[row] = -INFINITY;
        return;
    }
    if (nsplit <= 1) return;  // one CTA owned the whole segment and wrote the row itself

    constexpr int kRowF4 = D / 4;
    const bool col = lane < kRowF4;
    auto rec = [&](int sidx) { return sidx == 0 ? (int64_t)kind * p.part_cap + i_first : (int64_t)(i_first + sidx); };
    auto acc_ptr = [&](int sidx) {
        return reinterpret_cast<const float4 *>(p.part_acc + rec(sidx) * (kMaxGroup * D) + head * D) + lane;
    };
    auto state_ptr = [&](int sidx) { return reinterpret_cast<const float4 *>(p.part_state + rec(sidx) * kStateFloats + 8 * head); };

    // first batch of this warp's records: in flight before anything is waited for
    float4 a[kSmallBatch], st[kSmallBatch];
#pragma unroll
    for (int k = 0; k < kSmallBatch; ++k) {
        const int i = warp + kSmallStripes * k;
        a[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        st[k] = make_float4(-INFINITY, 0.f, 0.f, 0.f);
        if (i < nsplit) {
            if (col) a[k] = __ldcg(acc_ptr(i));
            st[k] = __ldcg(state_ptr(i));
        }
    }
    // the segment's maximum (every warp computes it: lane -> record)
    float M = -INFINITY;
#pragma unroll 1
    for (int i0 = 0; i0 < nsplit; i0 += 32)
        if (i0 + lane < nsplit) M = fmaxf(M, __ldcg(state_ptr(i0 + lane)).x);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(kFullMask, M, o));

    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
    float den = 0.f, den_x = 0.f;
    int i0 = warp;
    while (true) {
#pragma unroll
        for (int k = 0; k < kSmallBatch; ++k) {
            const float w = st[k].x == -INFINITY ? 0.f : ex2(st[k].x - M);  // empty split (R11): weight 0
            den += w * st[k].y;
            den_x += w * st[k].z;
            num.x += w * a[k].x; num.y += w * a[k].y; num.z += w * a[k].z; num.w += w * a[k].w;
        }
        i0 += kSmallStripes * kSmallBatch;
        if (i0 >= nsplit) break;
#pragma unroll
        for (int k = 0; k < kSmallBatch; ++k) {
            const int i = i0 + kSmallStripes * k;
            a[k] = make_float4(0.f, 0.f, 0.f, 0.f);
            st[k] = make_float4(-INFINITY, 0.f, 0.f, 0.f);
            if (i < nsplit) {
                if (col) a[k] = __ldcg(acc_ptr(i));
                st[k] = __ldcg(state_ptr(i));
            }
        }
    }
    if (col) *reinterpret_cast<float4 *>(&s_num[warp][4 * lane]) = num;
    if (lane == 0) { s_den[warp][0] = den; s_den[warp][1] = den_x; }
    __syncthreads();
    if (warp != 0) return;
    float d = s_den[0][0], dx = s_den[0][1];
    float4 n = num;
#pragma unroll
    for (int w = 1; w < kSmallStripes; ++w) {
        d += s_den[w][0];
        dx += s_den[w][1];
        if (col) {
            const float4 o = *reinterpret_cast<const float4 *>(&s_num[w][4 * lane]);
            n.x += o.x; n.y += o.y; n.z += o.z; n.w += o.w;
        }
    }
    const float inv = 1.f / d;
    if (col) {
        uint2 packed;
        packed.x = pack_bf16x2(n.x * inv, n.y * inv);
        packed.y = pack_bf16x2(n.z * inv, n.w * inv);
        *reinterpret_cast<uint2 *>(p.out + row * D + 4 * lane) = packed;
    }
    if (p.lse_out && lane == 0) p.lse_out[row] = (M + log2f(dx)) * 0.69314718055994530942f;
#ifdef COMEM_TRACE
    if (p.trace && tid == 0) p.trace[(1024 + blockIdx.x) * 16 + 2] = globaltimer_ns();
#endif
}

}  // namespace

cudaError_t launch_combine_small(const DecodeParams &p, int head_dim, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.batch * p.num_kv_heads * p.group);
    cfg.blockDim = dim3(kSmallThreads);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p.no_pdl ? 0 : 1;
    if (head_dim == 128) return cudaLaunchKernelEx(&cfg, combine_small_kernel<128>, p);
    return cudaLaunchKernelEx(&cfg, combine_small_kernel<64>, p);
}

cudaError_t launch_combine(const DecodeParams &p, int head_dim, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.batch * p.num_kv_heads);
    cfg.blockDim = dim3(kCombineThreads);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    static PerDeviceOnce once128, once64;
    if (head_dim == 128) {
        const cudaError_t e = set_max_smem_once(combine_kernel<128>, MergeCfg<128>::kStageBytes, once128);
        if (e != cudaSuccess) return e;
        cfg.dynamicSmemBytes = MergeCfg<128>::kStageBytes;
        return cudaLaunchKernelEx(&cfg, combine_kernel<128>, p);
    }
    const cudaError_t e = set_max_smem_once(combine_kernel<64>, MergeCfg<64>::kStageBytes, once64);
    if (e != cudaSuccess) return e;
    cfg.dynamicSmemBytes = MergeCfg<64>::kStageBytes;
    return cudaLaunchKernelEx(&cfg, combine_kernel<64>, p);
}

}  // namespace comem
