// prefill_params.cuh — kernel argument block and launcher of the paged causal prefill kernel (prefill_attn.cu).
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

namespace comem {

struct PrefillParams {
    const int32_t *block_table;  // [batch][max_pages]
    const int32_t *seq_lens;     // [batch]: tokens in the cache, the chunk's own tokens included
    const int32_t *q_start;      // [batch + 1]: rows of q / out that belong to each sequence
    __nv_bfloat16 *out;          // [total_q][Hq][D]
    float *lse_out;              // [total_q][Hq] or nullptr
    int batch;
    int num_q_heads;
    int num_kv_heads;
    int group;                   // G = Hq / Hkv
    int rows_per_tile;           // R = 128 / G query positions per 128-row tile
    int max_pages;
    int page_size;
    int page_tile_shift;         // log2(page_size / 16)
    float scale_log2;            // softmax_scale * log2(e)
};

// grid: an upper bound on the number of (sequence, kv head, tile pair) items; surplus CTAs exit at once
cudaError_t launch_prefill_attn(const CUtensorMap &tm_q, const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                                const PrefillParams &p, int head_dim, int grid, cudaStream_t stream, bool pdl);

}  // namespace comem
