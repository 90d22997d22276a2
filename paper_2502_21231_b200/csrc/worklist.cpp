// worklist.cpp — host builder of the attention work-item tables (see worklist.h).
#include "worklist.h"

#include <algorithm>
#include <map>
#include <new>

#ifndef BS_FWD_LONE_FIRST
#define BS_FWD_LONE_FIRST 1  // experiment switch
#endif

namespace bs {

namespace {
inline size_t align256(size_t x) { return (x + 255) & ~size_t(255); }
inline int32_t ceil_div(int64_t a, int64_t b) { return (int32_t)((a + b - 1) / b); }

struct Range {
  int32_t begin, end;
  bool operator<(const Range& o) const { return begin < o.begin; }
};

// Check that ranges (sorted by begin, duplicates removed) are pairwise disjoint and list the gaps
// of [lo,hi) they leave uncovered.
bs_status_t gaps_of(const std::vector<Range>& rs, int32_t lo, int32_t hi, const char* what,
                    SchedTables* out) {
  int32_t cur = lo;
  for (const Range& r : rs) {
    BS_REQUIRE(r.begin >= cur, BS_ERR_INVALID_ARG,
               "%s ranges of two segments overlap without being identical (at row %d)", what,
               r.begin);
    if (r.begin > cur) out->fill.push_back({cur, r.begin});
    cur = r.end;
  }
  if (cur < hi) out->fill.push_back({cur, hi});
  out->max_fill_rows = 0;
  for (const RowRange& f : out->fill)
    out->max_fill_rows = std::max<int64_t>(out->max_fill_rows, f.end - f.begin);
  return BS_OK;
}

bs_status_t check_seg(const bs_seg_t& g, int i, int32_t q_rows, int32_t kv_rows) {
  BS_REQUIRE(0 <= g.q_begin && g.q_begin < g.q_end && g.q_end <= q_rows, BS_ERR_INVALID_ARG,
             "segment %d: q range [%d,%d) empty or outside [0,%d)", i, g.q_begin, g.q_end, q_rows);
  BS_REQUIRE(0 <= g.k_begin && g.k_begin < g.k_end && g.k_end <= kv_rows, BS_ERR_INVALID_ARG,
             "segment %d: k range [%d,%d) empty or outside [0,%d)", i, g.k_begin, g.k_end, kv_rows);
  return BS_OK;
}

// Key b is visible to query a iff b <= a + off (a in [0, q_len), b in [0, k_len)).  Every offset
// >= k_len - 1 means "all keys" and every offset <= -q_len means "none", so the offset is stored
// clamped to [-q_len, k_len]: the mask is unchanged, and the kernels' 32-bit index arithmetic
// (row + offset) cannot overflow for callers who pass INT32_MAX / INT32_MIN as sentinels.
inline int32_t clamp_offset(int32_t off, int32_t q_len, int32_t k_len) {
  return std::max<int32_t>(-q_len, std::min<int32_t>(off, k_len));
}
}  // namespace

WsLayout ws_layout(size_t n_items, size_t n_spans, size_t n_groups, size_t n_fill, size_t tmap_bytes) {
  WsLayout L;
  L.items_off = sizeof(SchedHeader);
  L.spans_off = align256(L.items_off + n_items * sizeof(Item));
  L.groups_off = align256(L.spans_off + n_spans * sizeof(Span));
  L.fill_off = align256(L.groups_off + n_groups * sizeof(Group));
  L.tmaps_off = align256(L.fill_off + n_fill * sizeof(RowRange));
  L.total = align256(L.tmaps_off + tmap_bytes);
  return L;
}

namespace {
// index of `end_row` in `rows` (appended if new); `seen` maps end row -> index
int32_t clip_index(std::map<int32_t, int32_t>& seen, std::vector<int32_t>& rows, int32_t end_row) {
  auto it = seen.find(end_row);
  if (it != seen.end()) return it->second;
  const int32_t idx = (int32_t)rows.size();
  rows.push_back(end_row);
  seen.emplace(end_row, idx);
  return idx;
}
}  // namespace

size_t ws_upper_bound(int64_t rows, int32_t n_segs, bool bwd) {
  // items: every distinct range of length L yields ceil(L / tile) <= L / tile + 1 items
  const int64_t tile = bwd ? kTile : 2 * kTile;
  // forward: a range may add a lone first tile besides its last, partly filled item
  const size_t n_items = (size_t)(rows / tile + (bwd ? 1 : 2) * (int64_t)n_segs + 1);
  // clipped tensor maps: forward one (V) per key range; backward two per query range + two per key range
  const size_t tmap_bytes = (size_t)n_segs * (bwd ? 4 : 1) * kTensorMapBytes;
  return ws_layout(n_items, (size_t)n_segs, (size_t)n_segs, (size_t)n_segs + 1, tmap_bytes).total;
}

namespace {
// Order the groups by total cost (descending), the items of a group by cost (descending), and
// number the units: group-major, then head, then item.
bs_status_t finish_groups(std::vector<std::pair<int32_t, int32_t>>& group_items, int32_t n_heads,
                          SchedTables* out) {
  struct G {
    int32_t begin, n;
    int64_t cost;
  };
  std::vector<G> gs;
  for (auto& gi : group_items) {
    int64_t c = 0;
    for (int32_t i = gi.first; i < gi.first + gi.second; ++i) c += out->items[i].cost;
    gs.push_back({gi.first, gi.second, c});
  }
  std::stable_sort(gs.begin(), gs.end(), [](const G& a, const G& b) { return a.cost > b.cost; });
  std::vector<Item> sorted;
  sorted.reserve(out->items.size());
  int64_t units = 0;
  for (const G& g : gs) {
    const int32_t begin = (int32_t)sorted.size();
    sorted.insert(sorted.end(), out->items.begin() + g.begin, out->items.begin() + g.begin + g.n);
    std::stable_sort(sorted.begin() + begin, sorted.end(),
                     [](const Item& a, const Item& b) { return a.cost > b.cost; });
    BS_REQUIRE(units + (int64_t)g.n * n_heads <= INT32_MAX, BS_ERR_INVALID_ARG,
               "too many work units for one call");
    out->groups.push_back({begin, g.n, (int32_t)units, 0});
    units += (int64_t)g.n * n_heads;
  }
  out->items.swap(sorted);
  out->n_units = (int32_t)units;
  return BS_OK;
}
}  // namespace

bs_status_t build_fwd_tables(const bs_seg_t* segs, int32_t n_segs, int32_t q_rows, int32_t kv_rows,
                             int32_t out_begin, int32_t out_end, int32_t n_heads,
                             SchedTables* out) {
  try {
    std::vector<std::pair<int32_t, int32_t>> group_items;
    std::vector<int32_t> order(n_segs);
    for (int32_t i = 0; i < n_segs; ++i) {
      bs_status_t rc = check_seg(segs[i], i, q_rows, kv_rows);
      if (rc != BS_OK) return rc;
      BS_REQUIRE(segs[i].q_begin >= out_begin && segs[i].q_end <= out_end, BS_ERR_INVALID_ARG,
                 "segment %d: q range [%d,%d) outside the output rows [%d,%d)", i, segs[i].q_begin,
                 segs[i].q_end, out_begin, out_end);
      order[i] = i;
    }
    // group by q range; keep the caller's order inside a group
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
      return segs[a].q_begin != segs[b].q_begin ? segs[a].q_begin < segs[b].q_begin
                                                : segs[a].q_end < segs[b].q_end;
    });
    std::vector<Range> ranges;
    std::map<int32_t, int32_t> seen_span;
    for (int32_t i = 0; i < n_segs;) {
      const bs_seg_t& g0 = segs[order[i]];
      int32_t j = i;
      const int32_t span_begin = (int32_t)out->spans.size();
      while (j < n_segs && segs[order[j]].q_begin == g0.q_begin &&
             segs[order[j]].q_end == g0.q_end) {
        const bs_seg_t& g = segs[order[j]];
        const int32_t k_len = g.k_end - g.k_begin;
        out->spans.push_back({g.k_begin, k_len,
                              clamp_offset(g.causal_offset, g.q_end - g.q_begin, k_len),
                              k_len % kTile ? clip_index(seen_span, out->clip_span_rows, g.k_end) : -1});
        ++j;
      }
      ranges.push_back({g0.q_begin, g0.q_end});
      const int32_t q_len = g0.q_end - g0.q_begin;
      const int32_t first_item = (int32_t)out->items.size();
      // An item is two 128-row tiles that share the CTA (one TMEM slot each).  A range with an
      // odd number of tiles leaves one tile alone, and a lone tile runs at half the CTA's rate
      // for all of its key blocks: the lone one is the range's FIRST tile (the fewest visible
      // blocks under a causal mask), not its last (the most).  `limit` bounds the item's rows.
      auto emit = [&](int32_t a0, int32_t limit) {
        Item it{};
        it.row0 = g0.q_begin + a0;
        it.local0 = a0;
        it.range_len = limit;
        it.span_begin = span_begin;
        it.n_spans = j - i;
        int32_t cost = 0;
        for (int t = 0; t < 2; ++t) {
          const int32_t at = a0 + t * kTile;
          if (at >= limit) break;
          const int64_t a_last = std::min<int64_t>(at + kTile, limit) - 1;
          for (int32_t s = span_begin; s < span_begin + it.n_spans; ++s) {
            const int64_t vis = std::min<int64_t>(out->spans[s].len, a_last + out->spans[s].off + 1);
            if (vis > 0) it.tile_blocks[t] += (int32_t)ceil_div(vis, kTile);
          }
          cost += it.tile_blocks[t];
        }
        it.cost = cost;
        out->items.push_back(it);
      };
      const int32_t n_tiles = ceil_div(q_len, kTile);
      int32_t a0 = 0;
      if (BS_FWD_LONE_FIRST && n_tiles > 1 && n_tiles % 2 == 1) {
        emit(0, kTile);
        a0 = kTile;
      }
      for (; a0 < q_len; a0 += 2 * kTile) emit(a0, q_len);
      group_items.push_back({first_item, (int32_t)out->items.size() - first_item});
      i = j;
    }
    bs_status_t rc = finish_groups(group_items, n_heads, out);
    if (rc != BS_OK) return rc;
    std::sort(ranges.begin(), ranges.end());
    return gaps_of(ranges, out_begin, out_end, "query", out);
  } catch (const std::bad_alloc&) {
    return fail(BS_ERR_HOST_OOM, "out of host memory building the forward work list");
  }
}

bs_status_t build_bwd_tables(const bs_seg_t* segs, int32_t n_segs, int32_t q_rows, int32_t kv_rows,
                             int32_t n_heads, SchedTables* out) {
  try {
    std::vector<std::pair<int32_t, int32_t>> group_items;
    std::vector<int32_t> order(n_segs);
    for (int32_t i = 0; i < n_segs; ++i) {
      bs_status_t rc = check_seg(segs[i], i, q_rows, kv_rows);
      if (rc != BS_OK) return rc;
      order[i] = i;
    }
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
      return segs[a].k_begin != segs[b].k_begin ? segs[a].k_begin < segs[b].k_begin
                                                : segs[a].k_end < segs[b].k_end;
    });
    std::vector<Range> ranges;
    std::map<int32_t, int32_t> seen_span, seen_item;
    for (int32_t i = 0; i < n_segs;) {
      const bs_seg_t& g0 = segs[order[i]];
      int32_t j = i;
      const int32_t span_begin = (int32_t)out->spans.size();
      while (j < n_segs && segs[order[j]].k_begin == g0.k_begin &&
             segs[order[j]].k_end == g0.k_end) {
        const bs_seg_t& g = segs[order[j]];
        const int32_t q_len = g.q_end - g.q_begin;
        out->spans.push_back({g.q_begin, q_len,
                              clamp_offset(g.causal_offset, q_len, g.k_end - g.k_begin),
                              q_len % kTile ? clip_index(seen_span, out->clip_span_rows, g.q_end) : -1});
        ++j;
      }
      ranges.push_back({g0.k_begin, g0.k_end});
      const int32_t k_len = g0.k_end - g0.k_begin;
      group_items.push_back({(int32_t)out->items.size(), ceil_div(k_len, kTile)});
      for (int32_t b0 = 0; b0 < k_len; b0 += kTile) {
        Item it{};
        it.row0 = g0.k_begin + b0;
        it.local0 = b0;
        it.range_len = k_len;
        it.span_begin = span_begin;
        it.n_spans = j - i;
        it.tile_blocks[0] = b0 + kTile > k_len ? clip_index(seen_item, out->clip_item_rows, g0.k_end) : -1;
        int32_t cost = 0;
        for (int32_t s = span_begin; s < span_begin + it.n_spans; ++s) {
          // query a sees key b0 iff a >= b0 - off: query tiles from floor(a_min / tile) on
          const int64_t a_min = std::max<int64_t>(0, (int64_t)b0 - out->spans[s].off);
          if (a_min < out->spans[s].len)
            cost += ceil_div(out->spans[s].len, kTile) - (int32_t)(a_min / kTile);
        }
        it.cost = cost;
        out->items.push_back(it);
      }
      i = j;
    }
    bs_status_t rc = finish_groups(group_items, n_heads, out);
    if (rc != BS_OK) return rc;
    std::sort(ranges.begin(), ranges.end());
    return gaps_of(ranges, 0, kv_rows, "key", out);
  } catch (const std::bad_alloc&) {
    return fail(BS_ERR_HOST_OOM, "out of host memory building the backward work list");
  }
}

}  // namespace bs
