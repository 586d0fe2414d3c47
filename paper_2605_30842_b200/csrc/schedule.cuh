// schedule.cuh — the split-KV scheduler.
//
// Work unit: one TILE = 16 consecutive tokens of one (sequence b, kv head) pair.
// Tiles are linearised in (b, kv_head, tile) order; sequence b contributes
// T_b = ceil(L_b / 16) tiles per kv head, so the whole step is
// W = Hkv * sum_b T_b tiles.  The persistent grid's CTA i owns the contiguous
// range [floor(i*W/NC), floor((i+1)*W/NC)): every CTA streams the same number of
// bytes (+-1 tile) however ragged the batch is.  A CTA whose range covers a
// whole (b, kv_head) segment writes the final output row itself; a segment cut
// by a range boundary yields one partial per CTA that touches it (at most two
// partials per CTA: its first and its last segment), merged by the combine
// kernel in CTA-index order.
//
// Everything here is a function of (seq_lens, num_kv_heads, grid size) only:
// logical positions, never physical page ids, arrival order or atomics.  That
// is what makes the result bit-identical under page permutation.
#pragma once
#include <cstdint>

#ifdef __CUDACC__
#define COMEM_HD __host__ __device__ __forceinline__
#else
#define COMEM_HD inline
#endif

namespace comem {

constexpr int kTileTokens = 16;
constexpr int kTileShift = 4;
// Fewer than this many tiles per CTA is not worth a partial + combine round trip.
constexpr int kMinTilesPerCta = 16;
constexpr int kMaxGroup = 8;
// Largest batch the split kernel's shared-memory prefix table is sized for (== COMEM_MAX_BATCH).
constexpr int kMaxBatch = 4096;

COMEM_HD int tiles_of(int seq_len) { return seq_len <= 0 ? 0 : (seq_len + kTileTokens - 1) >> kTileShift; }

COMEM_HD int sched_num_ctas(int64_t total_tiles, int grid_ctas)
{
    int64_t want = (total_tiles + kMinTilesPerCta - 1) / kMinTilesPerCta;
    if (want < 1) want = 1;
    return want < grid_ctas ? (int)want : grid_ctas;
}

// first tile of CTA i (i in [0, nc]); cta_begin(nc) == total_tiles
COMEM_HD int64_t cta_begin(int i, int64_t total_tiles, int nc) { return ((int64_t)i * total_tiles) / nc; }

// the CTA whose range contains tile x (0 <= x < total_tiles)
COMEM_HD int cta_of_tile(int64_t x, int64_t total_tiles, int nc)
{
    return (int)(((x + 1) * nc - 1) / total_tiles);
}

// Split partials in the workspace.  A CTA writes at most two records: kind 0 for its FIRST segment,
// kind 1 for its LAST segment when that is a different one.  Structure of arrays, indexed [kind][cta]:
//   acc   fp32 [2][cap][8 heads][D]      un-normalised accumulator rows
//   state fp32 [2][cap][8 heads][8]      per head one 32-byte sector {m, l, lx, 0, 0, 0, 0, 0}
// A segment cut by CTAs i_first..i_last is therefore record (kind k0, i_first) followed by the
// CONTIGUOUS run (kind 0, i_first+1 .. i_last): the merge fetches it with two bulk copies.
constexpr int kStateFloats = 8 * kMaxGroup;
COMEM_HD int record_floats(int head_dim) { return kMaxGroup * head_dim; }

}  // namespace comem
