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

}  // namespace

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
