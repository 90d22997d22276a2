// worklist.h — work-item tables of the attention kernels (host-built, uploaded into the caller's
// workspace).  This is the single-device analogue of the paper's balance scheduler (Alg. 2,
// sort by cost descending, always feed the least-loaded worker): work units are
// ordered longest-first and pulled by persistent CTAs from one atomic cursor.
//
// Unit order (what the cursor walks): groups (= distinct ranges, most expensive first) x heads x
// the group's items (most expensive first).  All CTAs therefore work on a handful of (range, head)
// pairs at any time, whose K/V (forward) resp. Q/dO/dQ_acc (backward) rows stay in L2 while every
// tile of the pair is processed; the cheapest units of the cheapest range come last (short tail).
//
// Forward item  = up to 256 consecutive query rows (two 128-row MMA tiles) of one distinct query
//                 range; its spans are the key ranges of every segment on that query range
//                 (softmax over the union).  The kernel multiplies the item list by the Q heads.
//                 A range with an odd number of tiles gives its FIRST tile an item of its own
//                 (a lone tile runs at half the CTA's rate; under a causal mask the first tile
//                 has the fewest key blocks), then pairs.
// Backward item = one 128-key tile of one distinct key range; its spans are the query ranges of
//                 every segment on that key range.  The kernel multiplies the list by the KV heads
//                 and loops over the G query heads of the group and the visible query tiles.
#pragma once
#include <cstdint>
#include <vector>

#include "common.h"

namespace bs {

constexpr int kTile = 128;  // MMA tile edge in rows / keys
constexpr size_t kTensorMapBytes = 128;  // sizeof(CUtensorMap)

struct Span {     // forward: a key range;  backward: a query range
  int32_t begin;  // first row in the K/V (fwd) or Q (bwd) buffer
  int32_t len;    // rows
  int32_t off;    // key b visible to query a  iff  b <= a + off  (a, b local to their ranges)
  int32_t clip;   // index of the range end's clipped tensor maps (SchedTables::clip_span_rows),
                  // -1 if the range's length is a multiple of the tile (no ragged last tile)
};
struct Item {
  int32_t row0;        // first buffer row of the item (fwd: Q rows; bwd: K/V rows)
  int32_t local0;      // index of row0 inside its range (fwd: a0; bwd: b0)
  int32_t range_len;   // bwd: length of the key range; fwd: end of the item's rows inside its query
                       // range (the range length, or local0 + 128 for a lone first tile)
  int32_t span_begin;  // first span in the span table
  int32_t n_spans;
  int32_t cost;        // 128x128 blocks the item visits per head
  int32_t tile_blocks[2];  // fwd: of those, the blocks of Q tile 0 / 1; bwd: [0] = index of the
                           // clipped K / V tensor maps (SchedTables::clip_item_rows) if this is the
                           // ragged last tile of its key range, else -1
};
struct Group {           // the items of one distinct range; units = n_items x heads
  int32_t item_begin;    // first item in the item table
  int32_t n_items;
  int32_t unit_begin;    // first unit index of the group
  int32_t pad;
};
struct RowRange {
  int32_t begin, end;
};
struct SchedHeader {  // first 256 bytes of the workspace
  int32_t counter;    // dynamic scheduler cursor (zeroed by the upload)
  int32_t n_items, n_spans, n_fill;
  int32_t n_groups, n_units;
  int32_t pad[58];
};
static_assert(sizeof(SchedHeader) == 256, "header size");
static_assert(sizeof(Item) == 32 && sizeof(Span) == 16 && sizeof(Group) == 16, "table element sizes");

struct SchedTables {
  std::vector<Item> items;     // grouped by range; inside a group sorted by cost, descending
  std::vector<Span> spans;
  std::vector<Group> groups;   // sorted by total cost, descending
  int32_t n_units = 0;         // sum over groups of n_items x heads
  std::vector<RowRange> fill;  // rows of the output range covered by no item
  int64_t max_fill_rows = 0;
  // Range ends that are not tile-aligned: the ragged last tile of such a range is loaded through
  // a tensor map whose row extent stops at the end, so that TMA zero-fills the rows past it
  // (rows of another document, or uninitialised rows with NaN / Inf, never reach an MMA).
  std::vector<int32_t> clip_span_rows;  // end rows of the spans' ranges (fwd: K/V rows, bwd: Q rows)
  std::vector<int32_t> clip_item_rows;  // bwd: end rows of the key ranges (K/V rows)
  std::vector<uint8_t> tmaps;           // 128-byte CUtensorMap objects, filled by the entry point:
                                        // fwd [span clip] = V; bwd [2 i] = Q, [2 i + 1] = dO of
                                        // span clip i, then [2 j] = K, [2 j + 1] = V of item clip j
};

// Workspace layout: [SchedHeader][items][spans][groups][fill ranges][tensor maps], each 256-byte
// aligned.
struct WsLayout {
  size_t items_off, spans_off, groups_off, fill_off, tmaps_off, total;
};
WsLayout ws_layout(size_t n_items, size_t n_spans, size_t n_groups, size_t n_fill, size_t tmap_bytes);
// Upper bounds used by bs_attn_workspace_bytes (no segment list yet).
size_t ws_upper_bound(int64_t rows, int32_t n_segs, bool bwd);

// Forward: group segments by query range; rows [out_begin,out_end) not covered go to `fill`.
// n_heads = heads the kernel multiplies the item list by (Hq forward, Hkv backward).
bs_status_t build_fwd_tables(const bs_seg_t* segs, int32_t n_segs, int32_t q_rows, int32_t kv_rows,
                             int32_t out_begin, int32_t out_end, int32_t n_heads, SchedTables* out);
// Backward: group segments by key range; all kv_rows rows not covered go to `fill`.
bs_status_t build_bwd_tables(const bs_seg_t* segs, int32_t n_segs, int32_t q_rows, int32_t kv_rows,
                             int32_t n_heads, SchedTables* out);

}  // namespace bs
