// api.cu — the C ABI of libcomem_decode.so (include/comem_decode_attn.h): argument
// validation, TMA descriptor cache, workspace carving, launches.  No torch types, no device
// allocation, no CPU fallback: without a sm_100 device every compute entry point returns
// COMEM_ERR_CUDA / COMEM_ERR_UNSUPPORTED.
#include "../../include/comem_decode_attn.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "decode_params.cuh"
#include "prefill_params.cuh"
#include "schedule.cuh"

namespace comem {
namespace {

constexpr int kMaxGridCtas = 1024;  // workspace is sized for this many persistent CTAs
static_assert(kMaxGridCtas == kMaxGridCtasBound, "schedule.cuh's 32-bit fast paths assume this bound");
constexpr float kLog2e = 1.4426950408889634f;
constexpr int kPrefillMaxGroup = 16;  // a 128-row query tile holds 128 / G positions x G heads
static_assert(kMaxBatch == COMEM_MAX_BATCH, "header and scheduler disagree on the batch limit");

std::atomic<int> g_grid_override{0};
std::atomic<int> g_pdl{1};

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct WorkspaceLayout {
    size_t counters, flag, part_acc, part_state, q, new_k, new_v, out, lse, total;
};

WorkspaceLayout workspace_layout(int batch, int hq, int hkv, int d)
{
    WorkspaceLayout w;
    size_t off = 0;
    w.flag = off;      // comem_validate_inputs' verdict word: offset 0 whatever the shape
    off = align_up(off + sizeof(int), 256);
    w.counters = off;  // next, so that a buffer initialised for a large shape is initialised for smaller ones
    off = align_up(off + (size_t)batch * hkv * sizeof(int), 256);
    w.part_acc = off;
    off = align_up(off + (size_t)2 * kMaxGridCtas * record_floats(d) * sizeof(float), 256);
    w.part_state = off;
    off = align_up(off + (size_t)2 * kMaxGridCtas * kStateFloats * sizeof(float), 256);
    w.q = off;
    off = align_up(off + (size_t)batch * hq * d * 2, 256);
    w.new_k = off;
    off = align_up(off + (size_t)batch * hkv * d * 2, 256);
    w.new_v = off;
    off = align_up(off + (size_t)batch * hkv * d * 2, 256);
    w.out = off;
    off = align_up(off + (size_t)batch * hq * d * 2, 256);
    w.lse = off;
    off = align_up(off + (size_t)batch * hq * 4, 256);
    w.total = off;
    return w;
}

int check_shape(int hq, int hkv, int d, int ps, int batch, int max_pages, int64_t num_pages)
{
    if (batch <= 0 || hq <= 0 || hkv <= 0 || max_pages <= 0 || num_pages <= 0) return COMEM_ERR_INVALID_ARG;
    if (hq % hkv != 0) return COMEM_ERR_INVALID_ARG;
    const int g = hq / hkv;
    if (d != 64 && d != 128) return COMEM_ERR_UNSUPPORTED;
    if (ps != 16 && ps != 32) return COMEM_ERR_UNSUPPORTED;
    if (g < 1 || g > kMaxGroup) return COMEM_ERR_UNSUPPORTED;  // the group is packed into one 8-wide MMA dimension
    if (batch > COMEM_MAX_BATCH) return COMEM_ERR_UNSUPPORTED;
    // TMA row coordinate (page * page_size) and the linear tile count must fit in int32
    if (num_pages * ps >= (int64_t)1 << 31) return COMEM_ERR_UNSUPPORTED;
    if ((int64_t)batch * max_pages * (ps / kTileTokens) * hkv >= (int64_t)1 << 31) return COMEM_ERR_UNSUPPORTED;
    return COMEM_OK;
}

// ---- device capability (cached per device) ---------------------------------------------------
int check_device()
{
    static std::mutex mu;
    static int cached_dev = -1, cached_status = COMEM_ERR_CUDA;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(mu);
    if (dev == cached_dev) return cached_status;
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    cached_dev = dev;
    cached_status = (major == 10) ? COMEM_OK : COMEM_ERR_UNSUPPORTED;
    return cached_status;
}

// ---- TMA descriptors --------------------------------------------------------------------------
// The pool [P][ps][Hkv][D] is described to the TMA unit as a 4-D tensor
//   dim0 = 64 elements of d (128 B, the swizzle span)     stride 2 B
//   dim1 = P * ps token rows                               stride Hkv*D*2 B
//   dim2 = D / 64 halves of the head vector                stride 128 B
//   dim3 = Hkv                                             stride D*2 B
// with box {64, 16, D/64, 1}: one load brings a [16 tokens][D] tile of one kv head and lays
// it in shared memory as D/64 sub-tiles of [16 rows][128 B], 128-byte swizzled, which
// ldmatrix then reads without bank conflicts.
using EncodeFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                              const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                              CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                              CUtensorMapFloatOOBfill);

EncodeFn encode_fn()
{
    static EncodeFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            p = nullptr;
        }
        return reinterpret_cast<EncodeFn>(p);
    }();
    return fn;
}

struct MapKey {
    const void *ptr;
    int64_t num_pages;
    int ps, hkv, d, elem_bytes, hnd, box_rows;
    bool operator==(const MapKey &o) const
    {
        return ptr == o.ptr && num_pages == o.num_pages && ps == o.ps && hkv == o.hkv && d == o.d &&
               elem_bytes == o.elem_bytes && hnd == o.hnd && box_rows == o.box_rows;
    }
};
struct MapEntry {
    MapKey key;
    CUtensorMap map;
};

// FP8 pools (elem_bytes 1): a token row of one kv head is D bytes (128 B = the swizzle span at D 128; D 64: unswizzled), so
//   dim0 = 128 bytes of d, dim1 = P * ps token rows (stride Hkv*D B), dim2 = 1, dim3 = Hkv (stride D B),
// box {128, 16, 1, 1}: a [16 tokens][128 B] tile, 128-byte swizzled, read with 16-byte shared loads.
// HND layout [P][Hkv][ps][D]: dim1 = ps slots (stride D B), dim2 = Hkv (stride ps*D B), dim3 = P (stride Hkv*ps*D B).
// box_rows: token rows per box of the bf16 map: 16 (a whole tile, the decode kernels and the prefill kernel's V), or 8
// (the prefill kernel's K: half tiles, so that the 8-row groups of a 128-token block sit at one uniform pitch and
// S = Q K^T is one N = 128 instruction per k-step).
int get_tensor_map(const void *pool, int64_t num_pages, int ps, int hkv, int d, CUtensorMap *out, int elem_bytes = 2,
                   int hnd = 0, int box_rows = kTileTokens)
{
    static std::mutex mu;
    static std::vector<MapEntry> cache;
    static size_t next_evict = 0;
    const MapKey key{pool, num_pages, ps, hkv, d, elem_bytes, hnd, box_rows};
    std::lock_guard<std::mutex> lock(mu);
    for (const MapEntry &e : cache)
        if (e.key == key) { *out = e.map; return COMEM_OK; }
    EncodeFn enc = encode_fn();
    if (!enc) return COMEM_ERR_CUDA;
    const cuuint64_t gdim[4] = {64, (cuuint64_t)num_pages * ps, (cuuint64_t)(d / 64), (cuuint64_t)hkv};
    const cuuint64_t gstride[3] = {(cuuint64_t)hkv * d * 2, 128, (cuuint64_t)d * 2};
    const cuuint32_t box[4] = {64, (cuuint32_t)box_rows, (cuuint32_t)(d / 64), 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    MapEntry e;
    e.key = key;
    CUresult r;
    if (elem_bytes == 1) {
        cuuint64_t gdim8[4] = {(cuuint64_t)d, (cuuint64_t)num_pages * ps, 1, (cuuint64_t)hkv};
        cuuint64_t gstride8[3] = {(cuuint64_t)hkv * d, (cuuint64_t)d, (cuuint64_t)d};
        if (hnd) {
            gdim8[1] = (cuuint64_t)ps; gdim8[2] = (cuuint64_t)hkv; gdim8[3] = (cuuint64_t)num_pages;
            gstride8[0] = (cuuint64_t)d; gstride8[1] = (cuuint64_t)ps * d; gstride8[2] = (cuuint64_t)hkv * ps * d;
        }
        const cuuint32_t box8[4] = {(cuuint32_t)d, (cuuint32_t)kTileTokens, 1, 1};
        // D = 128: 128-byte rows, 128-byte swizzle; D = 64: plain 64-byte rows (decode_split.cu, Cfg)
        r = enc(&e.map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, const_cast<void *>(pool), gdim8, gstride8, box8, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, d == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                d == 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else {
        r = enc(&e.map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void *>(pool), gdim, gstride,
                box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                d == 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (r != CUDA_SUCCESS) return COMEM_ERR_CUDA;
    if (cache.size() < 64) cache.push_back(e);
    else { cache[next_evict] = e; next_evict = (next_evict + 1) % cache.size(); }
    *out = e.map;
    return COMEM_OK;
}

// Ragged query tensor q [total_q][Hq][D] of the prefill kernel, as a 4-D tensor
//   dim0 = 64 elements of d (128 B)   dim1 = Hq heads (stride D*2 B)   dim2 = total_q rows (stride Hq*D*2 B)
//   dim3 = D / 64 halves (stride 128 B)
// with box {64, G, R, D/64}: one load brings the G heads of one kv head's group for R consecutive query rows and lays
// them in shared memory as [D/64][R][G][128 B], 128-byte swizzled -- row (position * G + head) of a K-major
// tcgen05 A operand.  Rows past total_q are zero-filled.  Not cached: one encode per call (host arithmetic only).
int make_q_tensor_map(const void *q, int64_t total_q, int hq, int d, int group, int rows, CUtensorMap *out)
{
    EncodeFn enc = encode_fn();
    if (!enc) return COMEM_ERR_CUDA;
    const cuuint64_t gdim[4] = {64, (cuuint64_t)hq, (cuuint64_t)total_q, (cuuint64_t)(d / 64)};
    const cuuint64_t gstride[3] = {(cuuint64_t)d * 2, (cuuint64_t)hq * d * 2, 128};
    const cuuint32_t box[4] = {64, (cuuint32_t)group, (cuuint32_t)rows, (cuuint32_t)(d / 64)};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void *>(q), gdim, gstride, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? COMEM_OK : COMEM_ERR_CUDA;
}

constexpr int kMaxDevices = 64;

// Persistent-grid size: the call's own option, else the process default override, else one CTA per SM of the
// CURRENT device (cached per device ordinal).
int grid_for(int head_dim, int *grid, const comem_launch_opts *opts = nullptr)
{
    (void)head_dim;
    static std::mutex mu;
    static int cached[kMaxDevices] = {};
    const int ov = (opts && opts->grid_ctas > 0) ? opts->grid_ctas : g_grid_override.load();
    if (ov > 0) { *grid = ov < kMaxGridCtas ? ov : kMaxGridCtas; return COMEM_OK; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(mu);
    int uncached = 0;
    int &c = dev < kMaxDevices ? cached[dev] : uncached;
    if (c == 0) {
        int g = 0;
        if (split_default_grid(head_dim, &g) != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
        c = g < kMaxGridCtas ? g : kMaxGridCtas;
    }
    *grid = c;
    return COMEM_OK;
}

// programmatic stream serialization for this call: its own option (0 / 1), else the process default
bool pdl_for(const comem_launch_opts *opts)
{
    if (opts && opts->programmatic_launch >= 0) return opts->programmatic_launch != 0;
    return g_pdl.load() != 0;
}

#ifdef COMEM_TRACE
unsigned long long *g_trace = nullptr;
#endif

// Is this host pointer pinned AND mapped into the device address space?  If so return the device
// alias (identical under UVA, but ask anyway).
void *device_alias(const void *host_ptr)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, host_ptr) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (at.type != cudaMemoryTypeHost || at.devicePointer == nullptr) return nullptr;
    return at.devicePointer;
}

bool debug_validate()
{
    static const bool on = [] { const char *e = std::getenv("COMEM_DEBUG_VALIDATE"); return e && e[0] == '1'; }();
    return on;
}

// testing aid for the kernel's recovery paths (a schedule guess that fails its validation): see decode_split.cu
bool debug_stale_guess()
{
    static const bool on = [] { const char *e = std::getenv("COMEM_DEBUG_STALE_GUESS"); return e && e[0] == '1'; }();
    return on;
}

bool aligned(const void *p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

}  // namespace
}  // namespace comem

using namespace comem;

extern "C" {

int comem_version(void) { return 130; }

const char *comem_status_string(int status)
{
    switch (status) {
        case COMEM_OK: return "ok";
        case COMEM_ERR_INVALID_ARG: return "invalid argument";
        case COMEM_ERR_UNSUPPORTED: return "unsupported shape or device (needs sm_100; head_dim 64/128; page_size 16/32; group 1..8)";
        case COMEM_ERR_WORKSPACE: return "workspace missing or too small";
        case COMEM_ERR_CUDA: return "CUDA error (no device, driver entry point missing, or launch/execution failure)";
        default: return "unknown status";
    }
}

size_t comem_decode_attn_workspace_bytes(int batch, int num_q_heads, int num_kv_heads, int head_dim,
                                         int page_size, int max_pages_per_seq)
{
    (void)page_size;
    (void)max_pages_per_seq;
    if (batch <= 0 || num_q_heads <= 0 || num_kv_heads <= 0 || head_dim <= 0) return 0;
    return workspace_layout(batch, num_q_heads, num_kv_heads, head_dim).total;
}

int comem_workspace_init_async(void *workspace, size_t workspace_bytes, int batch, int num_q_heads,
                               int num_kv_heads, int head_dim, void *cuda_stream)
{
    if (batch <= 0 || num_q_heads <= 0 || num_kv_heads <= 0 || head_dim <= 0) return COMEM_ERR_INVALID_ARG;
    const WorkspaceLayout wl = workspace_layout(batch, num_q_heads, num_kv_heads, head_dim);
    if (!workspace || workspace_bytes < wl.total || !aligned(workspace, 256)) return COMEM_ERR_WORKSPACE;
    const int st = check_device();
    if (st != COMEM_OK) return st;
    if (cudaMemsetAsync(static_cast<char *>(workspace) + wl.flag, 0, wl.part_acc - wl.flag,
                        static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return COMEM_OK;
}

#ifdef COMEM_TRACE
int comem_set_trace(void *buf) { g_trace = static_cast<unsigned long long *>(buf); return COMEM_OK; }
#endif

static int validate_impl(const int32_t *block_table, const int32_t *seq_lens, int batch, int max_pages_per_seq,
                         int page_size, int64_t num_pages, void *workspace, size_t workspace_bytes,
                         void *cuda_stream, int extra_tokens)
{
    if (!block_table || !seq_lens || batch <= 0 || max_pages_per_seq <= 0 || page_size <= 0 || num_pages <= 0)
        return COMEM_ERR_INVALID_ARG;
    const WorkspaceLayout wl = workspace_layout(batch, 1, 1, 64);
    if (!workspace || workspace_bytes < wl.counters || !aligned(workspace, 256)) return COMEM_ERR_WORKSPACE;
    const int st = check_device();
    if (st != COMEM_OK) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int *flag = reinterpret_cast<int *>(static_cast<char *>(workspace) + wl.flag);
    int verdict = 0;
    if (launch_validate(block_table, seq_lens, batch, max_pages_per_seq, page_size, num_pages, flag, stream, extra_tokens) != cudaSuccess ||
        cudaMemcpyAsync(&verdict, flag, sizeof(int), cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
        cudaMemsetAsync(flag, 0, sizeof(int), stream) != cudaSuccess || cudaStreamSynchronize(stream) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return verdict == 0 ? COMEM_OK : COMEM_ERR_INVALID_ARG;
}

int comem_validate_inputs(const int32_t *block_table, const int32_t *seq_lens, int batch,
                          int max_pages_per_seq, int page_size, int64_t num_pages, void *workspace,
                          size_t workspace_bytes, void *cuda_stream)
{
    return validate_impl(block_table, seq_lens, batch, max_pages_per_seq, page_size, num_pages, workspace,
                         workspace_bytes, cuda_stream, 0);
}

int comem_set_grid_ctas(int n)
{
    g_grid_override.store(n > 0 ? n : 0);
    return COMEM_OK;
}

int comem_set_programmatic_launch(int enabled)
{
    g_pdl.store(enabled ? 1 : 0);
    return COMEM_OK;
}

int comem_sm_partition(double bytes_a, double bytes_b, int num_sms, int min_ctas, int *ctas_a, int *ctas_b)
{
    if (!ctas_a || !ctas_b || num_sms < 2 || !(bytes_a >= 0.0) || !(bytes_b >= 0.0) || !std::isfinite(bytes_a) ||
        !std::isfinite(bytes_b))
        return COMEM_ERR_INVALID_ARG;
    if (min_ctas < 1) min_ctas = 1;
    if (2 * min_ctas > num_sms) min_ctas = num_sms / 2;
    // shares proportional to the bytes each batch must stream (the path is HBM-bound and an SM pulls a fixed
    // rate), so both grids finish together; round to nearest, then keep at least min_ctas on each side
    const double tot = bytes_a + bytes_b;
    int a = tot > 0.0 ? (int)(bytes_a / tot * num_sms + 0.5) : num_sms / 2;
    if (a < min_ctas) a = min_ctas;
    if (a > num_sms - min_ctas) a = num_sms - min_ctas;
    *ctas_a = a;
    *ctas_b = num_sms - a;
    return COMEM_OK;
}

int comem_grid_ctas(int head_dim)
{
    if (head_dim != 64 && head_dim != 128) return -COMEM_ERR_UNSUPPORTED;
    const int st = check_device();
    if (st != COMEM_OK) return -st;
    int g = 0;
    const int r = grid_for(head_dim, &g);
    return r == COMEM_OK ? g : -r;
}

int comem_schedule_host(const int32_t *seq_lens_host, int batch, int num_kv_heads, int grid_ctas,
                        int64_t *tile_begin, int *num_ctas)
{
    if (!seq_lens_host || !tile_begin || !num_ctas || batch <= 0 || num_kv_heads <= 0 || grid_ctas <= 0)
        return COMEM_ERR_INVALID_ARG;
    std::vector<int> prefix(batch + 1, 0);
    for (int b = 0; b < batch; ++b) prefix[b + 1] = prefix[b] + tiles_of(seq_lens_host[b]);
    const int64_t total = (int64_t)prefix[batch] * num_kv_heads;
    if (total > 0 && batch * num_kv_heads <= kAlignedMaxSegs) {
        int e[kAlignedMaxSegs + 1];
        if (aligned_build(prefix.data(), batch, num_kv_heads, grid_ctas, e)) {  // segment-aligned variant
            *num_ctas = grid_ctas;
            for (int s = 0; s < batch * num_kv_heads; ++s) {
                const int b = s / num_kv_heads, kvh = s - b * num_kv_heads, T = prefix[b + 1] - prefix[b];
                const int64_t seg0 = (int64_t)num_kv_heads * prefix[b] + (int64_t)kvh * T;
                for (int i = e[s]; i < e[s + 1]; ++i) tile_begin[i] = aligned_cta_begin(seg0, T, i - e[s], e[s + 1] - e[s]);
            }
            tile_begin[grid_ctas] = total;
            return COMEM_OK;
        }
    }
    const int nc = total == 0 ? 0 : sched_num_ctas(total, grid_ctas);
    *num_ctas = nc;
    for (int i = 0; i <= nc; ++i) tile_begin[i] = nc ? cta_begin(i, total, nc) : 0;
    return COMEM_OK;
}

static int decode_attn_impl(const void *q, const void *k_pages, const void *v_pages,
                            const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                            int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                            void *out, int batch, int max_pages_per_seq, int64_t num_pages,
                            float *lse_out, void *workspace, size_t workspace_bytes,
                            void *cuda_stream, int phases, int window, int sink_tokens,
                            const comem_launch_opts *opts, const float *k_scale = nullptr,
                            const float *v_scale = nullptr, bool kv_fp8 = false, int kv_layout = COMEM_KV_LAYOUT_NHD,
                            const void *k_pages_host = nullptr, const void *v_pages_host = nullptr,
                            int64_t num_pages_host = 0)
{
    if (sink_tokens < 0) return COMEM_ERR_INVALID_ARG;
    // unknown launch-flag bits: rejected on the host before anything else is looked at
    if (opts && (opts->flags & ~(COMEM_LAUNCH_KV_PREFIX_IMMUTABLE | COMEM_LAUNCH_SPLIT_COMBINE | COMEM_LAUNCH_Q_STABLE |
                                 COMEM_LAUNCH_FP8_TENSOR)))
        return COMEM_ERR_INVALID_ARG;
    if (kv_fp8 && (!k_scale || !v_scale || !aligned(k_scale, 4) || !aligned(v_scale, 4))) return COMEM_ERR_INVALID_ARG;
    if (kv_layout != COMEM_KV_LAYOUT_NHD && !(kv_fp8 && kv_layout == COMEM_KV_LAYOUT_HND)) return COMEM_ERR_INVALID_ARG;
    if ((phases & ~(COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE)) != 0 || phases == 0) return COMEM_ERR_INVALID_ARG;
    if (!q || !k_pages || !v_pages || !block_table || !seq_lens || !out) return COMEM_ERR_INVALID_ARG;
    int st = check_shape(num_q_heads, num_kv_heads, head_dim, page_size, batch, max_pages_per_seq, num_pages);
    if (st != COMEM_OK) return st;
    if (!std::isfinite(softmax_scale) || softmax_scale < 0.f) return COMEM_ERR_INVALID_ARG;
    if (!aligned(q, 16) || !aligned(out, 16) || !aligned(k_pages, 128) || !aligned(v_pages, 128) ||
        !aligned(block_table, 4) || !aligned(seq_lens, 4) || (lse_out && !aligned(lse_out, 4)))
        return COMEM_ERR_INVALID_ARG;
    const WorkspaceLayout wl = workspace_layout(batch, num_q_heads, num_kv_heads, head_dim);
    if (!workspace || workspace_bytes < wl.total || !aligned(workspace, 256)) return COMEM_ERR_WORKSPACE;
    if ((st = check_device()) != COMEM_OK) return st;

    CUtensorMap tm_k, tm_v;
    const int elem_bytes = kv_fp8 ? 1 : 2;
    const int hnd = kv_layout == COMEM_KV_LAYOUT_HND ? 1 : 0;
    if ((st = get_tensor_map(k_pages, num_pages, page_size, num_kv_heads, head_dim, &tm_k, elem_bytes, hnd)) != COMEM_OK) return st;
    if ((st = get_tensor_map(v_pages, num_pages, page_size, num_kv_heads, head_dim, &tm_v, elem_bytes, hnd)) != COMEM_OK) return st;
    // second tier ("offloaded to CPU"): pools of the same layout in pinned, device-mapped host memory
    CUtensorMap tm_kh, tm_vh;
    const bool host_tier = k_pages_host != nullptr;
    if (host_tier) {
        if (kv_fp8 || !v_pages_host || num_pages_host <= 0 || phases != (COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE)) return COMEM_ERR_INVALID_ARG;
        if (num_pages_host * page_size >= (int64_t)1 << 31) return COMEM_ERR_UNSUPPORTED;
        const void *dk = device_alias(k_pages_host), *dv = device_alias(v_pages_host);
        if (!dk || !dv || !aligned(dk, 128) || !aligned(dv, 128)) return COMEM_ERR_INVALID_ARG;  // not pinned + mapped
        if ((st = get_tensor_map(dk, num_pages_host, page_size, num_kv_heads, head_dim, &tm_kh)) != COMEM_OK) return st;
        if ((st = get_tensor_map(dv, num_pages_host, page_size, num_kv_heads, head_dim, &tm_vh)) != COMEM_OK) return st;
    }

    DecodeParams p;
    p.host_tier = host_tier ? 1 : 0;
    p.debug_stale_guess = debug_stale_guess() ? 1 : 0;
    p.k_scale = kv_fp8 ? k_scale : nullptr;
    p.v_scale = kv_fp8 ? v_scale : nullptr;
    p.kv_hnd = hnd;
    p.no_pdl = pdl_for(opts) ? 0 : 1;
    p.q = static_cast<const __nv_bfloat16 *>(q);
    p.block_table = block_table;
    p.seq_lens = seq_lens;
    p.out = static_cast<__nv_bfloat16 *>(out);
    p.lse_out = lse_out;
    p.part_acc = reinterpret_cast<float *>(static_cast<char *>(workspace) + wl.part_acc);
    p.part_state = reinterpret_cast<float *>(static_cast<char *>(workspace) + wl.part_state);
    p.part_cap = kMaxGridCtas;
    p.seg_counters = reinterpret_cast<int *>(static_cast<char *>(workspace) + wl.counters);
    const int flags = opts ? opts->flags : 0;  // (validated at the top)
    // COMEM_LAUNCH_FP8_TENSOR: the tcgen05 split kernel of decode_fp8_tc.cu (FP8 cache, D = 128, no window, batch <= 1024)
    const bool fp8_tensor = (flags & COMEM_LAUNCH_FP8_TENSOR) != 0;
    if (fp8_tensor && (!kv_fp8 || phases != (COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE))) return COMEM_ERR_INVALID_ARG;
    // the small dependent combine serves steps of few segments only (elsewhere the fused merge costs nothing)
    const bool small_combine = phases == (COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE) && (flags & COMEM_LAUNCH_SPLIT_COMBINE) &&
                               batch * num_kv_heads <= kAlignedMaxSegs;
    const bool fused = phases == (COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE) && !small_combine && !fp8_tensor;
    p.fuse_combine = fused ? 1 : 0;
    p.kv_immutable = (flags & COMEM_LAUNCH_KV_PREFIX_IMMUTABLE) ? 1 : 0;
    p.q_stable = (flags & COMEM_LAUNCH_Q_STABLE) ? 1 : 0;  // (only acts together with KV_PREFIX_IMMUTABLE)
#ifdef COMEM_TRACE
    p.trace = g_trace;
#endif
    p.batch = batch;
    p.num_q_heads = num_q_heads;
    p.num_kv_heads = num_kv_heads;
    p.group = num_q_heads / num_kv_heads;
    p.max_pages = max_pages_per_seq;
    p.page_size = page_size;
    p.page_tile_shift = page_size == 32 ? 1 : 0;
    p.scale_log2 = softmax_scale * kLog2e;
    p.window = window > 0 ? window : 0;
    p.sinks = window > 0 ? sink_tokens : 0;
    if ((st = grid_for(head_dim, &p.grid_ctas, opts)) != COMEM_OK) return st;

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (fp8_tensor) {
        if (!fp8_tc_supported(p, head_dim)) return COMEM_ERR_UNSUPPORTED;
        const bool small = batch * num_kv_heads <= kAlignedMaxSegs;
        if (launch_decode_fp8_tc(tm_k, tm_v, p, stream) != cudaSuccess ||
            (small ? launch_combine_small(p, head_dim, stream) : launch_combine(p, head_dim, stream)) != cudaSuccess) {
            cudaGetLastError();
            return COMEM_ERR_CUDA;
        }
        return COMEM_OK;
    }
    if ((phases & COMEM_PHASE_SPLIT) &&
        launch_decode_split(tm_k, tm_v, p, head_dim, stream, kv_fp8, host_tier ? &tm_kh : nullptr,
                            host_tier ? &tm_vh : nullptr) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    if (small_combine) {
        if (launch_combine_small(p, head_dim, stream) != cudaSuccess) {
            cudaGetLastError();
            return COMEM_ERR_CUDA;
        }
        return COMEM_OK;
    }
    if (!fused && (phases & COMEM_PHASE_COMBINE) && launch_combine(p, head_dim, stream) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return COMEM_OK;
}

int comem_decode_attn_phases_async(const void *q, const void *k_pages, const void *v_pages,
                                   const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                                   int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                                   void *out, int batch, int max_pages_per_seq, int64_t num_pages,
                                   float *lse_out, void *workspace, size_t workspace_bytes,
                                   void *cuda_stream, int phases, const comem_launch_opts *opts)
{
    return decode_attn_impl(q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads, head_dim,
                            page_size, softmax_scale, out, batch, max_pages_per_seq, num_pages, lse_out,
                            workspace, workspace_bytes, cuda_stream, phases, 0, 0, opts);
}

int comem_decode_attn_window_async(const void *q, const void *k_pages, const void *v_pages,
                                   const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                                   int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                                   void *out, int batch, int max_pages_per_seq, int64_t num_pages,
                                   float *lse_out, void *workspace, size_t workspace_bytes,
                                   void *cuda_stream, int window, int sink_tokens, const comem_launch_opts *opts)
{
    return decode_attn_impl(q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads, head_dim,
                            page_size, softmax_scale, out, batch, max_pages_per_seq, num_pages, lse_out,
                            workspace, workspace_bytes, cuda_stream, COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE,
                            window, sink_tokens, opts);
}

int comem_decode_attn_fp8_async(const void *q, const void *k_pages, const void *v_pages, const float *k_scale,
                                const float *v_scale, const int32_t *block_table, const int32_t *seq_lens,
                                int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                                float softmax_scale, void *out, int batch, int max_pages_per_seq,
                                int64_t num_pages, float *lse_out, void *workspace, size_t workspace_bytes,
                                void *cuda_stream, int window, int sink_tokens, int kv_layout,
                                const comem_launch_opts *opts)
{
    return decode_attn_impl(q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads, head_dim,
                            page_size, softmax_scale, out, batch, max_pages_per_seq, num_pages, lse_out,
                            workspace, workspace_bytes, cuda_stream, COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE,
                            window, sink_tokens, opts, k_scale, v_scale, true, kv_layout);
}

int comem_decode_attn_async(const void *q, const void *k_pages, const void *v_pages,
                            const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                            int num_kv_heads, int head_dim, int page_size, float softmax_scale, void *out,
                            int batch, int max_pages_per_seq, int64_t num_pages, float *lse_out,
                            void *workspace, size_t workspace_bytes, void *cuda_stream,
                            const comem_launch_opts *opts)
{
    return comem_decode_attn_phases_async(q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads,
                                          head_dim, page_size, softmax_scale, out, batch, max_pages_per_seq,
                                          num_pages, lse_out, workspace, workspace_bytes, cuda_stream,
                                          COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE, opts);
}

// ---- comem_decode_attn_static_async: the decode step for callers that cannot allocate -------------------------------
// The scratch the step needs (arrival counters, split partials) lives in THIS file-scope device array instead of a
// caller-allocated workspace: COMEM_STATIC_SCRATCH_BYTES (12 MiB) on every GPU that loads the library, until exit.
// In host code `g_static_scratch` is only the symbol's host-side stand-in, never a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[COMEM_STATIC_SCRATCH_BYTES];

static int static_scratch_ptr(void **ptr)
{
    static std::atomic<void *> cache[64];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    const bool tracked = dev >= 0 && dev < 64;
    void *q = tracked ? cache[dev].load(std::memory_order_acquire) : nullptr;
    if (!q) {
        if (cudaGetSymbolAddress(&q, g_static_scratch) != cudaSuccess || !q) {
            cudaGetLastError();
            return COMEM_ERR_CUDA;
        }
        if (tracked) cache[dev].store(q, std::memory_order_release);
    }
    *ptr = q;
    return COMEM_OK;
}

size_t comem_static_scratch_bytes(void) { return COMEM_STATIC_SCRATCH_BYTES; }

int comem_decode_attn_static_async(const void *q, const void *k_pages, const void *v_pages,
                                   const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                                   int num_kv_heads, int head_dim, int page_size, float softmax_scale, void *out,
                                   int batch, int max_pages_per_seq, int64_t num_pages, float *lse_out,
                                   void *cuda_stream, const comem_launch_opts *opts)
{
    int st = check_shape(num_q_heads, num_kv_heads, head_dim, page_size, batch, max_pages_per_seq, num_pages);
    if (st != COMEM_OK) return st;
    const WorkspaceLayout wl = workspace_layout(batch, num_q_heads, num_kv_heads, head_dim);
    if (wl.total > (size_t)COMEM_STATIC_SCRATCH_BYTES) return COMEM_ERR_WORKSPACE;  // shape beyond the static scratch
    if ((st = check_device()) != COMEM_OK) return st;
    void *scratch = nullptr;
    if ((st = static_scratch_ptr(&scratch)) != COMEM_OK) return st;
    // every call shares the array and finds the previous call's contents: the arrival counters must start at zero
    // (a call that completed left them zero, one that was cut short did not)
    if (cudaMemsetAsync(static_cast<char *>(scratch) + wl.flag, 0, wl.part_acc - wl.flag,
                        static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return decode_attn_impl(q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads, head_dim, page_size,
                            softmax_scale, out, batch, max_pages_per_seq, num_pages, lse_out, scratch,
                            COMEM_STATIC_SCRATCH_BYTES, cuda_stream, COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE, 0, 0, opts);
}

int comem_decode_attn_offload_async(const void *q, const void *k_pages, const void *v_pages, const void *k_pages_host,
                                    const void *v_pages_host, const int32_t *block_table, const int32_t *seq_lens,
                                    int num_q_heads, int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                                    void *out, int batch, int max_pages_per_seq, int64_t num_pages,
                                    int64_t num_pages_host, float *lse_out, void *workspace, size_t workspace_bytes,
                                    void *cuda_stream, const comem_launch_opts *opts)
{
    if (!k_pages_host || !v_pages_host) return COMEM_ERR_INVALID_ARG;
    return decode_attn_impl(q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads, head_dim, page_size,
                            softmax_scale, out, batch, max_pages_per_seq, num_pages, lse_out, workspace, workspace_bytes,
                            cuda_stream, COMEM_PHASE_SPLIT | COMEM_PHASE_COMBINE, 0, 0, opts, nullptr, nullptr, false,
                            COMEM_KV_LAYOUT_NHD, k_pages_host, v_pages_host, num_pages_host);
}

int comem_pages_copy_async(const void *k_src, const void *v_src, void *k_dst, void *v_dst, const int32_t *src_ids,
                           const int32_t *dst_ids, int n_pages, size_t page_bytes, void *cuda_stream)
{
    if (!k_src || !v_src || !k_dst || !v_dst || !src_ids || !dst_ids || n_pages < 0 || page_bytes == 0 || page_bytes % 16)
        return COMEM_ERR_INVALID_ARG;
    if (n_pages == 0) return COMEM_OK;
    if (n_pages > 65535 * 1024) return COMEM_ERR_UNSUPPORTED;
    const int st = check_device();
    if (st != COMEM_OK) return st;
    // a pinned host pool is addressed through its device alias; a device pointer is used as it is
    auto resolve = [](const void *p) -> void * {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        if (at.type == cudaMemoryTypeHost) return at.devicePointer;
        if (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) return const_cast<void *>(p);
        return nullptr;  // pageable host memory
    };
    void *ks = resolve(k_src), *vs = resolve(v_src), *kd = resolve(k_dst), *vd = resolve(v_dst);
    if (!ks || !vs || !kd || !vd || !aligned(ks, 16) || !aligned(vs, 16) || !aligned(kd, 16) || !aligned(vd, 16))
        return COMEM_ERR_INVALID_ARG;
    if (launch_pages_copy(ks, vs, kd, vd, src_ids, dst_ids, n_pages, page_bytes,
                          static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return COMEM_OK;
}

int comem_prefill_attn_async(const void *q, const void *k_pages, const void *v_pages, const int32_t *block_table,
                             const int32_t *seq_lens, const int32_t *q_start, int num_q_heads, int num_kv_heads,
                             int head_dim, int page_size, float softmax_scale, void *out, int batch, int total_q,
                             int max_pages_per_seq, int64_t num_pages, float *lse_out, void *cuda_stream,
                             const comem_launch_opts *opts)
{
    if (!q || !k_pages || !v_pages || !block_table || !seq_lens || !q_start || !out) return COMEM_ERR_INVALID_ARG;
    if (batch <= 0 || total_q <= 0 || num_q_heads <= 0 || num_kv_heads <= 0 || max_pages_per_seq <= 0 || num_pages <= 0)
        return COMEM_ERR_INVALID_ARG;
    if (num_q_heads % num_kv_heads != 0) return COMEM_ERR_INVALID_ARG;
    const int g = num_q_heads / num_kv_heads;
    if (head_dim != 64 && head_dim != 128) return COMEM_ERR_UNSUPPORTED;
    if (page_size != 16 && page_size != 32) return COMEM_ERR_UNSUPPORTED;
    if (g > kPrefillMaxGroup || batch > COMEM_MAX_BATCH) return COMEM_ERR_UNSUPPORTED;
    if (num_pages * page_size >= (int64_t)1 << 31) return COMEM_ERR_UNSUPPORTED;
    if (!std::isfinite(softmax_scale) || softmax_scale < 0.f) return COMEM_ERR_INVALID_ARG;
    if (!aligned(q, 16) || !aligned(out, 16) || !aligned(k_pages, 128) || !aligned(v_pages, 128) ||
        !aligned(block_table, 4) || !aligned(seq_lens, 4) || !aligned(q_start, 4) || (lse_out && !aligned(lse_out, 4)))
        return COMEM_ERR_INVALID_ARG;
    int st = check_device();
    if (st != COMEM_OK) return st;

    PrefillParams p;
    p.block_table = block_table;
    p.seq_lens = seq_lens;
    p.q_start = q_start;
    p.out = static_cast<__nv_bfloat16 *>(out);
    p.lse_out = lse_out;
    p.batch = batch;
    p.num_q_heads = num_q_heads;
    p.num_kv_heads = num_kv_heads;
    p.group = g;
    p.rows_per_tile = 128 / g;
    p.max_pages = max_pages_per_seq;
    p.page_size = page_size;
    p.page_tile_shift = page_size == 32 ? 1 : 0;
    p.scale_log2 = softmax_scale * kLog2e;

    CUtensorMap tm_q, tm_k, tm_v;
    if ((st = make_q_tensor_map(q, total_q, num_q_heads, head_dim, g, p.rows_per_tile, &tm_q)) != COMEM_OK) return st;
    if ((st = get_tensor_map(k_pages, num_pages, page_size, num_kv_heads, head_dim, &tm_k, 2, 0, 8)) != COMEM_OK) return st;
    if ((st = get_tensor_map(v_pages, num_pages, page_size, num_kv_heads, head_dim, &tm_v)) != COMEM_OK) return st;
    // upper bound on sum_b ceil(n_b / 2R): the chunk lengths live on the device
    const int64_t pair_pos = 2 * (int64_t)p.rows_per_tile;
    const int64_t items = ((int64_t)total_q / pair_pos + (batch < total_q ? batch : total_q)) * num_kv_heads;
    if (items >= (int64_t)1 << 31) return COMEM_ERR_UNSUPPORTED;
    // default: one CTA per work item (the hardware scheduler balances them); with grid_ctas the kernel is persistent on
    // that many SMs and each CTA takes every grid_ctas-th item (the SM-partition policy of the k-step-off pipeline)
    int grid = (int)items;
    if (opts && opts->grid_ctas > 0 && opts->grid_ctas < grid) grid = opts->grid_ctas;
    const cudaError_t le = launch_prefill_attn(tm_q, tm_k, tm_v, p, head_dim, grid,
                                               static_cast<cudaStream_t>(cuda_stream), pdl_for(opts));
    if (le != cudaSuccess) {
        if (std::getenv("COMEM_DEBUG_ERRORS")) fprintf(stderr, "comem_prefill_attn_async: %s\n", cudaGetErrorString(le));
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return COMEM_OK;
}

int comem_decode_attn(const void *q, const void *k_pages, const void *v_pages, const int32_t *block_table,
                      const int32_t *seq_lens, int num_q_heads, int num_kv_heads, int head_dim,
                      int page_size, float softmax_scale, void *out, int batch, int max_pages_per_seq,
                      int64_t num_pages, float *lse_out, void *workspace, size_t workspace_bytes)
{
    if (debug_validate()) {
        const int v = comem_validate_inputs(block_table, seq_lens, batch, max_pages_per_seq, page_size, num_pages,
                                            workspace, workspace_bytes, nullptr);
        if (v != COMEM_OK) return v;
    }
    const int st = comem_decode_attn_async(q, k_pages, v_pages, block_table, seq_lens, num_q_heads,
                                           num_kv_heads, head_dim, page_size, softmax_scale, out, batch,
                                           max_pages_per_seq, num_pages, lse_out, workspace,
                                           workspace_bytes, nullptr, nullptr);
    if (st != COMEM_OK) return st;
    if (cudaStreamSynchronize(nullptr) != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    return COMEM_OK;
}

int comem_kv_append_async(void *k_pages, void *v_pages, const int32_t *block_table, int32_t *seq_lens,
                          const void *new_k, const void *new_v, int num_kv_heads, int head_dim,
                          int page_size, int batch, int max_pages_per_seq, void *cuda_stream)
{
    if (!k_pages || !v_pages || !block_table || !seq_lens || !new_k || !new_v) return COMEM_ERR_INVALID_ARG;
    if (batch <= 0 || num_kv_heads <= 0 || max_pages_per_seq <= 0) return COMEM_ERR_INVALID_ARG;
    if (head_dim != 64 && head_dim != 128) return COMEM_ERR_UNSUPPORTED;
    if (page_size != 16 && page_size != 32) return COMEM_ERR_UNSUPPORTED;
    if (!aligned(k_pages, 16) || !aligned(v_pages, 16) || !aligned(new_k, 16) || !aligned(new_v, 16))
        return COMEM_ERR_INVALID_ARG;
    const int st = check_device();
    if (st != COMEM_OK) return st;
    if (launch_kv_append(static_cast<__nv_bfloat16 *>(k_pages), static_cast<__nv_bfloat16 *>(v_pages),
                         block_table, seq_lens, static_cast<const __nv_bfloat16 *>(new_k),
                         static_cast<const __nv_bfloat16 *>(new_v), num_kv_heads * head_dim, page_size,
                         batch, max_pages_per_seq, static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return COMEM_OK;
}

int comem_kv_append_fp8_async(void *k_pages, void *v_pages, const float *k_scale, const float *v_scale,
                              const int32_t *block_table, int32_t *seq_lens, const void *new_k, const void *new_v,
                              int num_kv_heads, int head_dim, int page_size, int batch, int max_pages_per_seq,
                              int kv_layout, void *cuda_stream)
{
    if (!k_pages || !v_pages || !k_scale || !v_scale || !block_table || !seq_lens || !new_k || !new_v)
        return COMEM_ERR_INVALID_ARG;
    if (batch <= 0 || num_kv_heads <= 0 || max_pages_per_seq <= 0) return COMEM_ERR_INVALID_ARG;
    if (kv_layout != COMEM_KV_LAYOUT_NHD && kv_layout != COMEM_KV_LAYOUT_HND) return COMEM_ERR_INVALID_ARG;
    if (head_dim != 64 && head_dim != 128) return COMEM_ERR_UNSUPPORTED;
    if (page_size != 16 && page_size != 32) return COMEM_ERR_UNSUPPORTED;
    if (!aligned(k_pages, 16) || !aligned(v_pages, 16) || !aligned(new_k, 4) || !aligned(new_v, 4) ||
        !aligned(k_scale, 4) || !aligned(v_scale, 4))
        return COMEM_ERR_INVALID_ARG;
    const int st = check_device();
    if (st != COMEM_OK) return st;
    if (launch_kv_append_fp8(static_cast<uint8_t *>(k_pages), static_cast<uint8_t *>(v_pages), k_scale, v_scale,
                             block_table, seq_lens, static_cast<const __nv_bfloat16 *>(new_k),
                             static_cast<const __nv_bfloat16 *>(new_v), num_kv_heads, head_dim, page_size, batch,
                             max_pages_per_seq, kv_layout == COMEM_KV_LAYOUT_HND ? 1 : 0,
                             static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    return COMEM_OK;
}

int comem_decode_step_host(const void *q_host, const void *new_k_host, const void *new_v_host, void *k_pages,
                           void *v_pages, const int32_t *block_table, int32_t *seq_lens, int num_q_heads,
                           int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                           void *out_host, int batch, int max_pages_per_seq, int64_t num_pages,
                           float *lse_host, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!q_host || !out_host || ((new_k_host == nullptr) != (new_v_host == nullptr))) return COMEM_ERR_INVALID_ARG;
    int st = check_shape(num_q_heads, num_kv_heads, head_dim, page_size, batch, max_pages_per_seq, num_pages);
    if (st != COMEM_OK) return st;
    const WorkspaceLayout wl = workspace_layout(batch, num_q_heads, num_kv_heads, head_dim);
    if (!workspace || workspace_bytes < wl.total || !aligned(workspace, 256)) return COMEM_ERR_WORKSPACE;
    if ((st = check_device()) != COMEM_OK) return st;
    if (debug_validate()) {
        if (!block_table || !seq_lens) return COMEM_ERR_INVALID_ARG;
        st = validate_impl(block_table, seq_lens, batch, max_pages_per_seq, page_size, num_pages, workspace,
                           workspace_bytes, cuda_stream, new_k_host ? 1 : 0);
        if (st != COMEM_OK) return st;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    char *ws = static_cast<char *>(workspace);
    const size_t q_bytes = (size_t)batch * num_q_heads * head_dim * 2;
    const size_t kv_bytes = (size_t)batch * num_kv_heads * head_dim * 2;
    // Fast path: every host buffer is pinned and device-mapped (cudaHostAlloc / cudaHostRegister, what
    // torch's pin_memory() gives).  The kernels then move the step's bytes themselves: K3 reads the
    // q / k / v rows over the host link (staging q in the workspace), the attention kernel writes out
    // (and lse) straight into host memory -- 2 launches + 1 synchronize, no cudaMemcpyAsync.
    {
        void *dq = device_alias(q_host), *dout = device_alias(out_host);
        void *dk = new_k_host ? device_alias(new_k_host) : nullptr;
        void *dv = new_v_host ? device_alias(new_v_host) : nullptr;
        void *dlse = lse_host ? device_alias(lse_host) : nullptr;
        const bool mapped = dq && dout && (!new_k_host || (dk && dv)) && (!lse_host || dlse) &&
                            aligned(dq, 16) && aligned(dout, 16) && (!dk || (aligned(dk, 16) && aligned(dv, 16)));
        if (mapped) {
            if (!k_pages || !v_pages || !block_table || !seq_lens) return COMEM_ERR_INVALID_ARG;
            if (launch_kv_append(static_cast<__nv_bfloat16 *>(k_pages), static_cast<__nv_bfloat16 *>(v_pages),
                                 block_table, seq_lens, static_cast<const __nv_bfloat16 *>(dk),
                                 static_cast<const __nv_bfloat16 *>(dv), num_kv_heads * head_dim, page_size, batch,
                                 max_pages_per_seq, stream, static_cast<const __nv_bfloat16 *>(dq),
                                 reinterpret_cast<__nv_bfloat16 *>(ws + wl.q), num_q_heads * head_dim) != cudaSuccess) {
                cudaGetLastError();
                return COMEM_ERR_CUDA;
            }
            st = comem_decode_attn_async(ws + wl.q, k_pages, v_pages, block_table, seq_lens, num_q_heads,
                                         num_kv_heads, head_dim, page_size, softmax_scale, dout, batch,
                                         max_pages_per_seq, num_pages, static_cast<float *>(dlse), workspace,
                                         workspace_bytes, cuda_stream, nullptr);
            if (st != COMEM_OK) return st;
            if (cudaStreamSynchronize(stream) != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
            return COMEM_OK;
        }
    }
    bool ok = cudaMemcpyAsync(ws + wl.q, q_host, q_bytes, cudaMemcpyHostToDevice, stream) == cudaSuccess;
    if (ok && new_k_host) {
        ok = cudaMemcpyAsync(ws + wl.new_k, new_k_host, kv_bytes, cudaMemcpyHostToDevice, stream) == cudaSuccess &&
             cudaMemcpyAsync(ws + wl.new_v, new_v_host, kv_bytes, cudaMemcpyHostToDevice, stream) == cudaSuccess;
        if (ok) {
            st = comem_kv_append_async(k_pages, v_pages, block_table, seq_lens, ws + wl.new_k, ws + wl.new_v,
                                       num_kv_heads, head_dim, page_size, batch, max_pages_per_seq, cuda_stream);
            if (st != COMEM_OK) return st;
        }
    }
    if (!ok) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    st = comem_decode_attn_async(ws + wl.q, k_pages, v_pages, block_table, seq_lens, num_q_heads, num_kv_heads,
                                 head_dim, page_size, softmax_scale, ws + wl.out, batch, max_pages_per_seq,
                                 num_pages, lse_host ? reinterpret_cast<float *>(ws + wl.lse) : nullptr,
                                 workspace, workspace_bytes, cuda_stream, nullptr);
    if (st != COMEM_OK) return st;
    ok = cudaMemcpyAsync(out_host, ws + wl.out, q_bytes, cudaMemcpyDeviceToHost, stream) == cudaSuccess;
    if (ok && lse_host)
        ok = cudaMemcpyAsync(lse_host, ws + wl.lse, (size_t)batch * num_q_heads * 4, cudaMemcpyDeviceToHost,
                             stream) == cudaSuccess;
    if (!ok || cudaStreamSynchronize(stream) != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    return COMEM_OK;
}

int comem_decode_step_host_fp8(const void *q_host, const void *new_k_host, const void *new_v_host, void *k_pages,
                               void *v_pages, const float *k_scale, const float *v_scale, const int32_t *block_table,
                               int32_t *seq_lens, int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                               float softmax_scale, void *out_host, int batch, int max_pages_per_seq, int64_t num_pages,
                               float *lse_host, void *workspace, size_t workspace_bytes, void *cuda_stream, int kv_layout)
{
    if (!q_host || !out_host || !new_k_host || !new_v_host || !k_pages || !v_pages || !k_scale || !v_scale ||
        !block_table || !seq_lens)
        return COMEM_ERR_INVALID_ARG;
    if (kv_layout != COMEM_KV_LAYOUT_NHD && kv_layout != COMEM_KV_LAYOUT_HND) return COMEM_ERR_INVALID_ARG;
    int st = check_shape(num_q_heads, num_kv_heads, head_dim, page_size, batch, max_pages_per_seq, num_pages);
    if (st != COMEM_OK) return st;
    const WorkspaceLayout wl = workspace_layout(batch, num_q_heads, num_kv_heads, head_dim);
    if (!workspace || workspace_bytes < wl.total || !aligned(workspace, 256)) return COMEM_ERR_WORKSPACE;
    if ((st = check_device()) != COMEM_OK) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    char *ws = static_cast<char *>(workspace);
    const size_t q_bytes = (size_t)batch * num_q_heads * head_dim * 2;
    const size_t kv_bytes = (size_t)batch * num_kv_heads * head_dim * 2;
    const int hnd = kv_layout == COMEM_KV_LAYOUT_HND ? 1 : 0;
    void *dq = device_alias(q_host), *dout = device_alias(out_host), *dk = device_alias(new_k_host),
         *dv = device_alias(new_v_host), *dlse = lse_host ? device_alias(lse_host) : nullptr;
    const bool mapped = dq && dout && dk && dv && (!lse_host || dlse) && aligned(dq, 16) && aligned(dout, 16) &&
                        aligned(dk, 4) && aligned(dv, 4);
    const void *nk = dk, *nv = dv;
    const void *q_src = dq;
    void *out_dst = dout;
    float *lse_dst = static_cast<float *>(dlse);
    bool ok = true;
    if (!mapped) {  // pageable host memory: the copy engine stages the rows
        ok = cudaMemcpyAsync(ws + wl.new_k, new_k_host, kv_bytes, cudaMemcpyHostToDevice, stream) == cudaSuccess &&
             cudaMemcpyAsync(ws + wl.new_v, new_v_host, kv_bytes, cudaMemcpyHostToDevice, stream) == cudaSuccess &&
             cudaMemcpyAsync(ws + wl.out, q_host, q_bytes, cudaMemcpyHostToDevice, stream) == cudaSuccess;
        if (!ok) { cudaGetLastError(); return COMEM_ERR_CUDA; }
        nk = ws + wl.new_k;
        nv = ws + wl.new_v;
        q_src = ws + wl.out;  // (staged to wl.q by the append kernel like the mapped path; wl.out is free until the attention runs)
        out_dst = ws + wl.out;
        lse_dst = lse_host ? reinterpret_cast<float *>(ws + wl.lse) : nullptr;
    }
    // K3 (FP8): quantise + append the new row with the page's scales, bump seq_lens, stage q in the workspace
    if (launch_kv_append_fp8(static_cast<uint8_t *>(k_pages), static_cast<uint8_t *>(v_pages), k_scale, v_scale,
                             block_table, seq_lens, static_cast<const __nv_bfloat16 *>(nk),
                             static_cast<const __nv_bfloat16 *>(nv), num_kv_heads, head_dim, page_size, batch,
                             max_pages_per_seq, hnd, stream, static_cast<const __nv_bfloat16 *>(q_src),
                             reinterpret_cast<__nv_bfloat16 *>(ws + wl.q), num_q_heads * head_dim) != cudaSuccess) {
        cudaGetLastError();
        return COMEM_ERR_CUDA;
    }
    st = comem_decode_attn_fp8_async(ws + wl.q, k_pages, v_pages, k_scale, v_scale, block_table, seq_lens, num_q_heads,
                                     num_kv_heads, head_dim, page_size, softmax_scale, out_dst, batch, max_pages_per_seq,
                                     num_pages, lse_dst, workspace, workspace_bytes, cuda_stream, 0, 0, kv_layout, nullptr);
    if (st != COMEM_OK) return st;
    if (!mapped) {
        ok = cudaMemcpyAsync(out_host, ws + wl.out, q_bytes, cudaMemcpyDeviceToHost, stream) == cudaSuccess;
        if (ok && lse_host)
            ok = cudaMemcpyAsync(lse_host, ws + wl.lse, (size_t)batch * num_q_heads * 4, cudaMemcpyDeviceToHost, stream) == cudaSuccess;
    }
    if (!ok || cudaStreamSynchronize(stream) != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    return COMEM_OK;
}

}  // extern "C"
