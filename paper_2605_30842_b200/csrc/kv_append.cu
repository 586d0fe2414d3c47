// kv_append.cu — K3: K_cache^(t) = [K_cache^(t-1); K^(t)], V likewise (typo
// corrected per DESIGN.md reading R3).  One CTA per sequence copies the new token's
// [Hkv][D] K row and V row (contiguous in the paged layout) into slot seq_len % page_size of
// page block_table[b][seq_len / page_size] with 16-byte stores, then bumps seq_lens[b].
// The same CTA can also stage sequence b's query rows (q_src -> q_dst, 16-byte copies): on the
// end-to-end path (comem_decode_step_host) new_k / new_v / q_src are device-mapped PINNED HOST
// pointers, so this one kernel is the whole host->device leg of a step (zero-copy reads over the
// host link) instead of three cudaMemcpyAsync calls.
#include "decode_params.cuh"
#include "ptx.cuh"

namespace comem {

namespace {

__global__ void __launch_bounds__(128)
kv_append_kernel(__nv_bfloat16 *k_pages, __nv_bfloat16 *v_pages, const int32_t *block_table,
                 int32_t *seq_lens, const __nv_bfloat16 *new_k, const __nv_bfloat16 *new_v,
                 int row_elems, int page_size, int max_pages, const __nv_bfloat16 *q_src,
                 __nv_bfloat16 *q_dst, int q_row_elems)
{
    // let the attention kernel queued behind this one start its prologue now (it computes its schedule
    // speculatively and re-validates after ITS griddepcontrol.wait, which still waits for this grid to finish)
    pdl_launch_dependents();
    pdl_wait_prior_grid();
    const int b = blockIdx.x;
    if (q_src != nullptr) {
        const uint4 *s = reinterpret_cast<const uint4 *>(q_src + (int64_t)b * q_row_elems);
        uint4 *d = reinterpret_cast<uint4 *>(q_dst + (int64_t)b * q_row_elems);
        for (int i = threadIdx.x; i < q_row_elems / 8; i += blockDim.x) d[i] = s[i];
    }
    if (new_k == nullptr) return;
    const int t = seq_lens[b];
    const int page = t / page_size;
    const int slot = t - page * page_size;
    // a full (or corrupt) row: the next table entry would be another sequence's -- append nothing, bump nothing
    if (t < 0 || page >= max_pages) return;
    const int64_t pid = block_table[(int64_t)b * max_pages + page];
    const int64_t dst = (pid * page_size + slot) * (int64_t)row_elems;
    const int vecs = row_elems / 8;  // uint4 = 8 bf16
    const uint4 *sk = reinterpret_cast<const uint4 *>(new_k + (int64_t)b * row_elems);
    const uint4 *sv = reinterpret_cast<const uint4 *>(new_v + (int64_t)b * row_elems);
    uint4 *dk = reinterpret_cast<uint4 *>(k_pages + dst);
    uint4 *dv = reinterpret_cast<uint4 *>(v_pages + dst);
    for (int i = threadIdx.x; i < vecs; i += blockDim.x) {
        dk[i] = sk[i];
        dv[i] = sv[i];
    }
    __syncthreads();  // every thread has read seq_lens[b] before it changes
    if (threadIdx.x == 0) seq_lens[b] = t + 1;
}

// FP8 cache (reading R18): the new token's bf16 rows are quantised with the scales of the page they land in,
//   byte = e4m3_rne_satfinite((float)x / scale[pid][kv head])      (IEEE fp32 quotient, then cvt.rn.satfinite)
// one CTA per sequence, one thread per pair of elements; then seq_lens[b] += 1.  hnd: pools [P][Hkv][ps][D].
__global__ void __launch_bounds__(128)
kv_append_fp8_kernel(uint8_t *k_pages, uint8_t *v_pages, const float *k_scale, const float *v_scale,
                     const int32_t *block_table, int32_t *seq_lens, const __nv_bfloat16 *new_k,
                     const __nv_bfloat16 *new_v, int num_kv_heads, int head_dim, int page_size, int max_pages, int hnd,
                     const __nv_bfloat16 *q_src, __nv_bfloat16 *q_dst, int q_row_elems)
{
    pdl_launch_dependents();  // as in kv_append_kernel
    pdl_wait_prior_grid();
    const int b = blockIdx.x;
    if (q_src != nullptr) {  // end-to-end path: stage sequence b's query rows (q_src may be pinned host memory)
        const uint4 *s = reinterpret_cast<const uint4 *>(q_src + (int64_t)b * q_row_elems);
        uint4 *d = reinterpret_cast<uint4 *>(q_dst + (int64_t)b * q_row_elems);
        for (int i = threadIdx.x; i < q_row_elems / 8; i += blockDim.x) d[i] = s[i];
    }
    const int t = seq_lens[b];
    const int page = t / page_size;
    const int slot = t - page * page_size;
    if (t < 0 || page >= max_pages) return;  // as in kv_append_kernel
    const int64_t pid = block_table[(int64_t)b * max_pages + page];
    const int row_elems = num_kv_heads * head_dim;
    const uint32_t *sk = reinterpret_cast<const uint32_t *>(new_k + (int64_t)b * row_elems);
    const uint32_t *sv = reinterpret_cast<const uint32_t *>(new_v + (int64_t)b * row_elems);
    for (int i = threadIdx.x; i < row_elems / 2; i += blockDim.x) {
        const int h = (2 * i) / head_dim, d = 2 * i - h * head_dim;
        const int64_t dst = (hnd ? (pid * num_kv_heads + h) * page_size + slot
                                 : (pid * page_size + slot) * num_kv_heads + h) * (int64_t)head_dim + d;
        const float ks = k_scale[pid * num_kv_heads + h], vs = v_scale[pid * num_kv_heads + h];
        const uint32_t kw = sk[i], vw = sv[i];
        uint16_t kq, vq;
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(kq)
            : "f"(__fdiv_rn(bf16hi_to_f32(kw), ks)), "f"(__fdiv_rn(bf16lo_to_f32(kw), ks)));
        asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(vq)
            : "f"(__fdiv_rn(bf16hi_to_f32(vw), vs)), "f"(__fdiv_rn(bf16lo_to_f32(vw), vs)));
        *reinterpret_cast<uint16_t *>(k_pages + dst) = kq;
        *reinterpret_cast<uint16_t *>(v_pages + dst) = vq;
    }
    __syncthreads();  // every thread has read seq_lens[b] before it changes
    if (threadIdx.x == 0) seq_lens[b] = t + 1;
}

// Debug aid (comem_validate_inputs): one CTA per sequence checks what the hot path trusts --
// seq_len within the table row's reach and every USED table entry a page id inside the pool.
// flag: 0 = fine; otherwise 1 + index of the first offending sequence seen.
__global__ void __launch_bounds__(128)
validate_kernel(const int32_t *block_table, const int32_t *seq_lens, int max_pages, int page_size,
                long long num_pages, int *flag, int extra_tokens)
{
    const int b = blockIdx.x;
    const int len = seq_lens[b] + extra_tokens;  // extra_tokens = 1: the state after the append about to run
    bool bad = seq_lens[b] < 0 || (long long)len > (long long)max_pages * page_size;
    if (!bad) {
        const int used = (len + page_size - 1) / page_size;
        for (int j = threadIdx.x; j < used; j += blockDim.x) {
            const int pid = block_table[(long long)b * max_pages + j];
            bad = bad || pid < 0 || pid >= num_pages;
        }
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicCAS(flag, 0, b + 1);
}

// comem_pages_copy_async: CTA (i, t) copies page src_ids[i] -> dst_ids[i] of the K pool (t = 0) or the V pool (t = 1)
// with 16-byte accesses; either side may be pinned host memory (zero-copy over the host link).
__global__ void __launch_bounds__(256)
pages_copy_kernel(const uint4 *k_src, const uint4 *v_src, uint4 *k_dst, uint4 *v_dst, const int32_t *src_ids,
                  const int32_t *dst_ids, size_t page_vecs)
{
    pdl_wait_prior_grid();
    const int i = blockIdx.x;
    const uint4 *src = (blockIdx.y ? v_src : k_src) + (size_t)src_ids[i] * page_vecs;
    uint4 *dst = (blockIdx.y ? v_dst : k_dst) + (size_t)dst_ids[i] * page_vecs;
    for (size_t e = threadIdx.x; e < page_vecs; e += blockDim.x) dst[e] = src[e];
}

}  // namespace

cudaError_t launch_pages_copy(const void *k_src, const void *v_src, void *k_dst, void *v_dst, const int32_t *src_ids,
                              const int32_t *dst_ids, int n_pages, size_t page_bytes, cudaStream_t stream)
{
    pages_copy_kernel<<<dim3(n_pages, 2), 256, 0, stream>>>(
        static_cast<const uint4 *>(k_src), static_cast<const uint4 *>(v_src), static_cast<uint4 *>(k_dst),
        static_cast<uint4 *>(v_dst), src_ids, dst_ids, page_bytes / 16);
    return cudaGetLastError();
}

cudaError_t launch_validate(const int32_t *block_table, const int32_t *seq_lens, int batch, int max_pages,
                            int page_size, int64_t num_pages, int *flag, cudaStream_t stream, int extra_tokens)
{
    cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), stream);
    if (e != cudaSuccess) return e;
    validate_kernel<<<batch, 128, 0, stream>>>(block_table, seq_lens, max_pages, page_size, (long long)num_pages, flag, extra_tokens);
    return cudaGetLastError();
}

cudaError_t launch_kv_append_fp8(uint8_t *k_pages, uint8_t *v_pages, const float *k_scale, const float *v_scale,
                                 const int32_t *block_table, int32_t *seq_lens, const __nv_bfloat16 *new_k,
                                 const __nv_bfloat16 *new_v, int num_kv_heads, int head_dim, int page_size, int batch,
                                 int max_pages, int hnd, cudaStream_t stream, const __nv_bfloat16 *q_src,
                                 __nv_bfloat16 *q_dst, int q_row_elems)
{
    kv_append_fp8_kernel<<<batch, 128, 0, stream>>>(k_pages, v_pages, k_scale, v_scale, block_table, seq_lens, new_k,
                                                   new_v, num_kv_heads, head_dim, page_size, max_pages, hnd, q_src, q_dst,
                                                   q_row_elems);
    return cudaGetLastError();
}

cudaError_t launch_kv_append(__nv_bfloat16 *k_pages, __nv_bfloat16 *v_pages, const int32_t *block_table,
                             int32_t *seq_lens, const __nv_bfloat16 *new_k, const __nv_bfloat16 *new_v,
                             int row_elems, int page_size, int batch, int max_pages, cudaStream_t stream,
                             const __nv_bfloat16 *q_src, __nv_bfloat16 *q_dst, int q_row_elems)
{
    kv_append_kernel<<<batch, 128, 0, stream>>>(k_pages, v_pages, block_table, seq_lens, new_k, new_v,
                                               row_elems, page_size, max_pages, q_src, q_dst, q_row_elems);
    return cudaGetLastError();
}

}  // namespace comem
