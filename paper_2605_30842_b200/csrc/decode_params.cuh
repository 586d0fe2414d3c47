// decode_params.cuh — kernel argument block shared by the split and combine launchers.
#pragma once
#include <atomic>
#include <cstdint>
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

namespace comem {

struct DecodeParams {
    const __nv_bfloat16 *q;      // [batch][Hq][D]
    const int32_t *block_table;  // [batch][max_pages]
    const int32_t *seq_lens;     // [batch]
    __nv_bfloat16 *out;          // [batch][Hq][D]
    float *lse_out;              // [batch][Hq] or nullptr
    float *part_acc;             // workspace: [2 kinds][part_cap][8][D] (schedule.cuh)
    float *part_state;           // workspace: [2 kinds][part_cap][8][8]
    int part_cap;                // records per kind the workspace holds (>= grid_ctas)
    int *seg_counters;           // workspace: [batch][Hkv] arrival counters, zero between launches
    int fuse_combine;            // 1: the last CTA to finish a cut segment merges it inside K1
#ifdef COMEM_TRACE
    unsigned long long *trace;   // development builds only: [grid][8] %globaltimer stamps per CTA
#endif
    int batch;
    int num_q_heads;
    int num_kv_heads;
    int group;                   // Hq / Hkv
    int max_pages;               // block-table row length
    int page_size;               // 16 or 32
    int page_tile_shift;         // log2(page_size / 16): tiles per page
    int grid_ctas;               // persistent grid size the schedule was sized for
    float scale_log2;            // softmax_scale * log2(e)
    int window;                  // sliding window in tokens (<= 0: none), schedule.cuh win_tiles
    int sinks;                   // attention-sink tokens kept at the start of every sequence
    const float *k_scale;        // FP8 cache only (reading R18): fp32 [P][Hkv] page scales, else nullptr
    const float *v_scale;
    int no_pdl;                  // host-side only: launch without programmatic stream serialization (comem_set_programmatic_launch)
    int kv_immutable;            // COMEM_LAUNCH_KV_PREFIX_IMMUTABLE: the caller promises that nothing still running when this
                                 // grid starts writes K/V rows (or their block-table entries / page scales) below each
                                 // sequence's last 16-token tile, so the ring may be filled before griddepcontrol.wait
    int q_stable;                // COMEM_LAUNCH_Q_STABLE: ... nor q: the consumers may start before the wait too
    int debug_stale_guess;       // COMEM_DEBUG_STALE_GUESS=1 (testing aid): the speculative schedule is computed from stale lengths
    int host_tier;               // a second pool in pinned host memory is addressed by block-table entries < 0 (bf16 only)
    int kv_hnd;                  // FP8 cache only: pools laid out [P][Hkv][ps][D] (a tile is 2 KiB contiguous) instead of [P][ps][Hkv][D]
};

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a per-DEVICE setting: remember, per kernel instantiation,
// the device ordinals it has been applied on (a process may drive the agent model on one GPU and the memory
// model on another).
struct PerDeviceOnce {
    std::atomic<unsigned char> done[64];
};
template <typename Kernel>
inline cudaError_t set_max_smem_once(Kernel kernel, int bytes, PerDeviceOnce &once)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && once.done[dev].load(std::memory_order_acquire)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && tracked) once.done[dev].store(1, std::memory_order_release);
    return e;
}

// launchers (defined in decode_split.cu / combine.cu / kv_append.cu)
// kv_fp8: the pools hold E4M3 bytes and p.k_scale / p.v_scale are set
cudaError_t launch_decode_split(const CUtensorMap &tm_k, const CUtensorMap &tm_v,
                                const DecodeParams &p, int head_dim, cudaStream_t stream, bool kv_fp8 = false,
                                const CUtensorMap *tm_k_host = nullptr, const CUtensorMap *tm_v_host = nullptr);
// FP8 cache with both contractions on tcgen05 (decode_fp8_tc.cu; COMEM_LAUNCH_FP8_TENSOR): the split kernel only, partial
// records as launch_decode_split writes them with fuse_combine == 0
bool fp8_tc_supported(const DecodeParams &p, int head_dim);
cudaError_t launch_decode_fp8_tc(const CUtensorMap &tm_k, const CUtensorMap &tm_v, const DecodeParams &p, cudaStream_t stream);
cudaError_t launch_combine(const DecodeParams &p, int head_dim, cudaStream_t stream);
// the small dependent combine (COMEM_LAUNCH_SPLIT_COMBINE; batch * Hkv <= kAlignedMaxSegs)
cudaError_t launch_combine_small(const DecodeParams &p, int head_dim, cudaStream_t stream);
cudaError_t launch_kv_append(__nv_bfloat16 *k_pages, __nv_bfloat16 *v_pages,
                             const int32_t *block_table, int32_t *seq_lens,
                             const __nv_bfloat16 *new_k, const __nv_bfloat16 *new_v, int row_elems,
                             int page_size, int batch, int max_pages, cudaStream_t stream,
                             const __nv_bfloat16 *q_src = nullptr, __nv_bfloat16 *q_dst = nullptr,
                             int q_row_elems = 0);
cudaError_t launch_kv_append_fp8(uint8_t *k_pages, uint8_t *v_pages, const float *k_scale, const float *v_scale,
                                 const int32_t *block_table, int32_t *seq_lens, const __nv_bfloat16 *new_k,
                                 const __nv_bfloat16 *new_v, int num_kv_heads, int head_dim, int page_size, int batch,
                                 int max_pages, int hnd, cudaStream_t stream, const __nv_bfloat16 *q_src = nullptr,
                                 __nv_bfloat16 *q_dst = nullptr, int q_row_elems = 0);
cudaError_t launch_pages_copy(const void *k_src, const void *v_src, void *k_dst, void *v_dst, const int32_t *src_ids,
                              const int32_t *dst_ids, int n_pages, size_t page_bytes, cudaStream_t stream);
cudaError_t launch_validate(const int32_t *block_table, const int32_t *seq_lens, int batch, int max_pages,
                            int page_size, int64_t num_pages, int *flag, cudaStream_t stream, int extra_tokens = 0);
// occupancy-derived persistent grid for the split kernel on the current device
cudaError_t split_default_grid(int head_dim, int *grid_ctas);
size_t split_smem_bytes(int head_dim, int batch);

}  // namespace comem
