// combine.cu — K2, the log-sum-exp combine.
//
// One CTA per output row (sequence b, query head h).  It recomputes the same schedule as the split kernel
// (schedule.cuh) to learn which CTAs cut this segment, then merges their fp32 partials
// (acc, m, l, lx) in CTA-index order (l sums the bf16-rounded p and normalises out; lx sums the
// unrounded p and only feeds lse_out):
//     M = max_s m_s;  w_s = 2^(m_s - M);  out = (sum_s w_s acc_s) / (sum_s w_s l_s)
// Segments owned by a single CTA were already written by the split kernel and are skipped;
// empty sequences (seq_len == 0) get +0.0 rows and lse = -inf here (reading R9).
#include "decode_params.cuh"
#include "ptx.cuh"
#include "schedule.cuh"

namespace comem {

namespace {

constexpr int kCombineThreads = 128;
constexpr int kParts = 4;  // split-index stripes summed in parallel, then merged in stripe order

template <int D>
__global__ void __launch_bounds__(kCombineThreads)
combine_kernel(const DecodeParams p)
{
    constexpr int kVec = D / 4;  // float4 lanes covering one row: 32 (D=128) / 16 (D=64)
    static_assert(kCombineThreads / kVec >= kParts, "layout");
    __shared__ int s_before, s_total;
    __shared__ float s_m[kCombineThreads / 32];
    __shared__ float s_den[kParts], s_denx[kParts];
    __shared__ float4 s_red[kParts][kVec];

    const int b = blockIdx.x / p.num_q_heads;
    const int h = blockIdx.x - b * p.num_q_heads;
    const int kvh = h / p.group;
    const int g = h - kvh * p.group;
    const int tid = threadIdx.x;
    const int64_t row = (int64_t)b * p.num_q_heads + h;

    if (tid == 0) { s_before = 0; s_total = 0; }
    __syncthreads();
    pdl_wait_prior_grid();  // seq_lens / partials may come from the kernels launched just before

    // tiles before sequence b, and in total (block reduction over seq_lens)
    {
        int before = 0, total = 0;
        for (int i = tid; i < p.batch; i += kCombineThreads) {
            const int ti = tiles_of(p.seq_lens[i]);
            total += ti;
            if (i < b) before += ti;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            before += __shfl_xor_sync(0xffffffffu, before, o);
            total += __shfl_xor_sync(0xffffffffu, total, o);
        }
        if ((tid & 31) == 0) { atomicAdd(&s_before, before); atomicAdd(&s_total, total); }
    }
    __syncthreads();
    pdl_launch_dependents();

    const int T = tiles_of(p.seq_lens[b]);
    if (T == 0) {
        for (int e = tid; e < D; e += kCombineThreads) p.out[row * D + e] = __float2bfloat16_rn(0.f);
        if (p.lse_out && tid == 0) p.lse_out[row] = -INFINITY;
        return;
    }
    const int64_t total = (int64_t)p.num_kv_heads * s_total;
    const int nc = sched_num_ctas(total, p.grid_ctas);
    const int64_t seg0 = (int64_t)p.num_kv_heads * s_before + (int64_t)kvh * T;
    const int64_t seg1 = seg0 + T;
    const int i_first = cta_of_tile(seg0, total, nc);
    const int i_last = cta_of_tile(seg1 - 1, total, nc);
    if (i_first == i_last) return;  // one CTA owned the whole segment and wrote the row itself
    const int nsplit = i_last - i_first + 1;
    const int stride = partial_stride_floats(D);
    // slot of split s: CTA i's first-segment slot (2i) unless the segment starts inside CTA i_first
    const int first_slot = 2 * i_first + (cta_begin(i_first, total, nc) < seg0 ? 1 : 0);
    auto slot_of = [&](int s) { return s == 0 ? first_slot : 2 * (i_first + s); };

    // pass A: M = max_s m_s
    float M = -INFINITY;
    for (int s = tid; s < nsplit; s += kCombineThreads)
        M = fmaxf(M, p.partials[(int64_t)slot_of(s) * stride + kMaxGroup * D + g]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    if ((tid & 31) == 0) s_m[tid >> 5] = M;
    __syncthreads();
    M = fmaxf(fmaxf(s_m[0], s_m[1]), fmaxf(s_m[2], s_m[3]));

    // pass B: kParts stripes of splits (s = part, part + kParts, ...) summed in parallel
    const int vec = tid % kVec;
    const int part = tid / kVec;
    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
    float den = 0.f, den_x = 0.f;
    if (part < kParts) {
#pragma unroll 4
        for (int s = part; s < nsplit; s += kParts) {
            const float *rec = p.partials + (int64_t)slot_of(s) * stride;
            const float w = ex2(rec[kMaxGroup * D + g] - M);
            const float4 a = *reinterpret_cast<const float4 *>(rec + g * D + 4 * vec);
            den += w * rec[kMaxGroup * D + kMaxGroup + g];
            den_x += w * rec[kMaxGroup * D + 2 * kMaxGroup + g];
            num.x += w * a.x; num.y += w * a.y; num.z += w * a.z; num.w += w * a.w;
        }
        s_red[part][vec] = num;
        if (vec == 0) { s_den[part] = den; s_denx[part] = den_x; }
    }
    __syncthreads();
    if (part == 0) {  // merge the stripes in stripe order
        float4 r = s_red[0][vec];
        float dsum = s_den[0], dxsum = s_denx[0];
#pragma unroll
        for (int q = 1; q < kParts; ++q) {
            const float4 o = s_red[q][vec];
            r.x += o.x; r.y += o.y; r.z += o.z; r.w += o.w;
            dsum += s_den[q];
            dxsum += s_denx[q];
        }
        const float inv = 1.f / dsum;
        __nv_bfloat162 lo = __floats2bfloat162_rn(r.x * inv, r.y * inv);
        __nv_bfloat162 hi = __floats2bfloat162_rn(r.z * inv, r.w * inv);
        uint2 packed;
        packed.x = *reinterpret_cast<uint32_t *>(&lo);
        packed.y = *reinterpret_cast<uint32_t *>(&hi);
        *reinterpret_cast<uint2 *>(p.out + row * D + 4 * vec) = packed;
        if (p.lse_out && vec == 0) p.lse_out[row] = (M + log2f(dxsum)) * 0.69314718055994530942f;
    }
}

}  // namespace

cudaError_t launch_combine(const DecodeParams &p, int head_dim, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.batch * p.num_q_heads);
    cfg.blockDim = dim3(kCombineThreads);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (head_dim == 128) return cudaLaunchKernelEx(&cfg, combine_kernel<128>, p);
    return cudaLaunchKernelEx(&cfg, combine_kernel<64>, p);
}

}  // namespace comem
