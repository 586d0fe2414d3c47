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

// ---- sliding window + attention sinks (reading R17) ---------------------------------
// The query sits at position L-1 and attends t < sinks or t >= L - window.  Only the tiles that
// hold a kept token are scheduled and read: the sink tiles [0, sink_tiles) and the window tiles
// [win_first, tiles_of(L)); a sequence's tile index j (0 <= j < total) maps to a logical tile through
// win_logical_tile.  window <= 0 or >= L: everything is kept and the map is the identity.
struct WinTiles {
    int sink_tiles, win_first, total;
    int lo, sk;  // kept tokens: t < sk or t >= lo (sk = min(sinks, lo))
};
COMEM_HD WinTiles win_tiles(int L, int window, int sinks)
{
    WinTiles w;
    const int all = tiles_of(L);
    w.lo = (window <= 0 || window >= L) ? 0 : L - window;
    w.sk = sinks < w.lo ? (sinks > 0 ? sinks : 0) : w.lo;
    w.win_first = w.lo >> kTileShift;
    const int st = (w.sk + kTileTokens - 1) >> kTileShift;
    w.sink_tiles = st < w.win_first ? st : w.win_first;
    w.total = L <= 0 ? 0 : w.sink_tiles + (all - w.win_first);
    return w;
}
COMEM_HD int seq_tiles(int L, int window, int sinks) { return window <= 0 ? tiles_of(L) : win_tiles(L, window, sinks).total; }
COMEM_HD int win_logical_tile(const WinTiles &w, int j) { return j < w.sink_tiles ? j : j - w.sink_tiles + w.win_first; }
// bit i set <=> token 16*tile + i is kept and < L
COMEM_HD unsigned win_alive_mask(const WinTiles &w, int L, int tile)
{
    const int base = tile << kTileShift;
    auto low = [](int n) -> unsigned { return n <= 0 ? 0u : (n >= kTileTokens ? 0xffffu : (1u << n) - 1u); };
    return low(L - base) & (low(w.sk - base) | (~low(w.lo - base) & 0xffffu));
}

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

// ---- segment-aligned variant -----------------------------------------------------------------
// A CTA whose linear range straddles a segment boundary pays for a second epilogue (S6) in
// mid-stream -- about 2 us, which a short step (one 32K sequence: ~18 us of streaming) cannot
// amortise, and which lands on the critical path because that CTA is then the last to arrive on
// its second segment.  When the step has FEW LONG segments the CTAs are therefore dealt to the
// segments instead: segment s (s = b * Hkv + kv head, in linear order) owns the CTAs
// [e[s], e[s+1]) with e[s+1] = round(tiles up to the end of s * grid / total tiles), and CTA j of
// its c owns tiles [j*T/c, (j+1)*T/c) of it.  No CTA sees two segments; the price is that c is the
// ideal share rounded, i.e. up to T/c - total/grid extra tiles on the slowest CTA.  The variant
// is used iff every non-empty segment gets a CTA and that price is below kAlignedMaxLossTiles
// (same decision, same integer arithmetic, in K1, K2 and comem_schedule_host).
constexpr int kAlignedMaxSegs = 64;
constexpr int kMaxGridCtasBound = 1024;  // j <= c <= grid <= 1024 (api.cu's kMaxGridCtas)
constexpr int kAlignedMaxLossTiles = 6;

COMEM_HD int aligned_boundary(int64_t tiles_to_end, int64_t total_tiles, int grid_ctas)
{
    // same value either way; the 32-bit form keeps 64-bit divisions off the launch's critical path
    if (total_tiles <= (int64_t)((0x7fffffff / 2) / grid_ctas))  // (a 32-bit division: grid_ctas is an int)
        return (int)(((uint32_t)tiles_to_end * (uint32_t)grid_ctas + (uint32_t)total_tiles / 2u) / (uint32_t)total_tiles);
    return (int)((tiles_to_end * grid_ctas + total_tiles / 2) / total_tiles);
}
// tiles on the busiest CTA if the work were cut evenly
COMEM_HD int ideal_tiles_per_cta(int64_t total_tiles, int grid_ctas)
{
    if (total_tiles <= 0x7fffffff - kMaxGridCtasBound)  // same value; keeps a 64-bit division off the launch's critical path
        return (int)(((uint32_t)total_tiles + (uint32_t)grid_ctas - 1u) / (uint32_t)grid_ctas);
    return (int)((total_tiles + grid_ctas - 1) / grid_ctas);
}
// is a segment of T tiles that was dealt c CTAs acceptable?
COMEM_HD bool aligned_segment_ok(int T, int c, int ideal)
{
    if (T == 0) return true;
    if (c < 1) return false;
    return (T + c - 1) / c - ideal <= kAlignedMaxLossTiles;
}
// Serial builder (host, K2): prefix[b] = tiles of sequences < b (batch + 1 entries).  Fills
// e[0 .. batch*hkv] and returns true iff the aligned variant applies.
COMEM_HD bool aligned_build(const int *prefix, int batch, int hkv, int grid_ctas, int *e)
{
    const int S = batch * hkv;
    const int64_t total = (int64_t)hkv * prefix[batch];
    if (S > kAlignedMaxSegs || total < (int64_t)grid_ctas * kMinTilesPerCta) return false;
    const int ideal = ideal_tiles_per_cta(total, grid_ctas);
    bool ok = true;
    e[0] = 0;
    for (int s = 0; s < S; ++s) {
        const int b = s / hkv, kvh = s - b * hkv;
        const int T = prefix[b + 1] - prefix[b];
        e[s + 1] = aligned_boundary((int64_t)hkv * prefix[b] + (int64_t)(kvh + 1) * T, total, grid_ctas);
        ok = ok && aligned_segment_ok(T, e[s + 1] - e[s], ideal);
    }
    return ok;
}
// first tile (linear coordinates) of CTA j of the c CTAs of a segment that starts at seg0 with T tiles
COMEM_HD int64_t aligned_cta_begin(int64_t seg0, int T, int j, int c)
{
    if (T <= 0x7fffffff / kMaxGridCtasBound) return seg0 + (int)((uint32_t)(j * T) / (uint32_t)c);
    return seg0 + ((int64_t)j * T) / c;
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
