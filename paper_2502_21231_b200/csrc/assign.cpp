// assign.cpp — bs_assign: the naive HDP solution (Algorithm 1; routine at
// PAPER.md:262) with offload ratio r = 0, host integers only.  The step directly upstream of
// bs_plan: a global batch of sequence lengths becomes, for every HDP rank and every round of the
// step, the bs_seq_t list that rank hands to bs_plan.  Readings R1-R4: include/bytescale_attn.h.
#include <algorithm>
#include <map>
#include <new>
#include <vector>

#include "common.h"

struct bs_assign_s {
  std::vector<int32_t> d;  // D(s_i)
  int32_t n_rounds = 0;
  std::vector<bs_seq_t> seqs;  // all micro-batches, back to back
  std::vector<int32_t> src;
  std::vector<bs_microbatch_t> mbs;  // sorted by (round, rank); pointers set last
};

namespace {

struct Pending {  // a micro-batch group before its round is known
  int32_t ranks;      // consecutive ranks it needs in one round
  int32_t seq_begin;  // its sequences in the flat arrays (a long sequence: one entry)
  int32_t seq_end;
  int32_t round, first_rank;
};

}  // namespace

extern "C" {

bs_status_t bs_assign(const int32_t* lens, int32_t n, int32_t capacity, int32_t d_hdp,
                      bs_assign_t** out) {
  BS_REQUIRE(out != nullptr, BS_ERR_INVALID_ARG, "bs_assign: out is null");
  *out = nullptr;
  BS_REQUIRE(n >= 0 && (lens != nullptr || n == 0), BS_ERR_INVALID_ARG, "bs_assign: bad lens / n");
  BS_REQUIRE(capacity >= 1 && d_hdp >= 1, BS_ERR_INVALID_ARG,
             "bs_assign: capacity %d and d_hdp %d must be positive", capacity, d_hdp);
  try {
    bs_assign_s* a = new bs_assign_s;
    struct Guard {
      bs_assign_s* p;
      ~Guard() { delete p; }
    } guard{a};
    a->d.resize(n);
    // lines 1-6: D(s_i) = ceil(s_i / C) (Eq. 3 with r = 0, Act linear); D = 1 goes to the pack list
    std::multimap<int32_t, int32_t, std::greater<int32_t>> pack;  // length (descending) -> index
    std::vector<int32_t> longs;
    for (int32_t i = 0; i < n; ++i) {
      BS_REQUIRE(lens[i] >= 1, BS_ERR_INVALID_ARG, "bs_assign: sequence %d has length %d", i, lens[i]);
      const int64_t d = ((int64_t)lens[i] + capacity - 1) / capacity;
      BS_REQUIRE(d <= d_hdp, BS_ERR_INVALID_ARG,
                 "bs_assign: sequence %d (%d tokens) needs %lld ranks of capacity %d, d_hdp is %d", i,
                 lens[i], (long long)d, capacity, d_hdp);
      a->d[i] = (int32_t)d;
      if (d == 1)
        pack.emplace(lens[i], i);  // equal lengths keep input order (multimap insertion order)
      else
        longs.push_back(i);
    }
    std::vector<Pending> groups;
    // long sequences first, in input order (line 10 places them before the bins, R4)
    for (int32_t i : longs) {
      const int32_t b = (int32_t)a->seqs.size();
      a->seqs.push_back({lens[i], a->d[i], 0});
      a->src.push_back(i);
      groups.push_back({a->d[i], b, b + 1, 0, 0});
    }
    // lines 7-9: one bin per pass; the longest remaining sequence that still fits, until none does
    while (!pack.empty()) {
      int32_t room = capacity;
      const int32_t b = (int32_t)a->seqs.size();
      for (;;) {
        auto it = pack.lower_bound(room);  // first key <= room in descending order
        if (it == pack.end()) break;
        room -= it->first;
        a->seqs.push_back({it->first, 1, 0});
        a->src.push_back(it->second);
        pack.erase(it);
      }
      groups.push_back({1, b, (int32_t)a->seqs.size(), 0, 0});
    }
    // line 10: first round with enough free ranks; ranks of a round are handed out from 0 upwards
    std::vector<int32_t> used;  // ranks taken in each round
    for (Pending& g : groups) {
      size_t k = 0;
      while (k < used.size() && d_hdp - used[k] < g.ranks) ++k;
      if (k == used.size()) used.push_back(0);
      g.round = (int32_t)k;
      g.first_rank = used[k];
      used[k] += g.ranks;
    }
    a->n_rounds = (int32_t)used.size();
    // one micro-batch per (round, rank): a long sequence becomes D shards with cp ranks 0..D-1
    std::vector<bs_seq_t> flat;
    std::vector<int32_t> flat_src;
    struct Slot {
      int32_t round, rank, begin, end;
    };
    std::vector<Slot> slots;
    for (const Pending& g : groups) {
      if (g.ranks > 1) {
        for (int32_t j = 0; j < g.ranks; ++j) {
          bs_seq_t s = a->seqs[g.seq_begin];
          s.rank = j;
          slots.push_back({g.round, g.first_rank + j, (int32_t)flat.size(), (int32_t)flat.size() + 1});
          flat.push_back(s);
          flat_src.push_back(a->src[g.seq_begin]);
        }
      } else {
        slots.push_back({g.round, g.first_rank, (int32_t)flat.size(),
                         (int32_t)flat.size() + (g.seq_end - g.seq_begin)});
        flat.insert(flat.end(), a->seqs.begin() + g.seq_begin, a->seqs.begin() + g.seq_end);
        flat_src.insert(flat_src.end(), a->src.begin() + g.seq_begin, a->src.begin() + g.seq_end);
      }
    }
    std::sort(slots.begin(), slots.end(), [](const Slot& x, const Slot& y) {
      return x.round != y.round ? x.round < y.round : x.rank < y.rank;
    });
    a->seqs.swap(flat);
    a->src.swap(flat_src);
    a->mbs.reserve(slots.size());
    for (const Slot& s : slots)
      a->mbs.push_back({s.round, s.rank, s.end - s.begin, a->seqs.data() + s.begin,
                        a->src.data() + s.begin});
    guard.p = nullptr;
    *out = a;
    return BS_OK;
  } catch (const std::bad_alloc&) {
    return bs::fail(BS_ERR_HOST_OOM, "bs_assign: out of host memory");
  }
}

int32_t bs_assign_n_rounds(const bs_assign_t* a) { return a ? a->n_rounds : 0; }
int32_t bs_assign_n_seqs(const bs_assign_t* a) { return a ? (int32_t)a->d.size() : 0; }
const int32_t* bs_assign_ranks_needed(const bs_assign_t* a) { return a ? a->d.data() : nullptr; }
int32_t bs_assign_n_microbatches(const bs_assign_t* a) { return a ? (int32_t)a->mbs.size() : 0; }
const bs_microbatch_t* bs_assign_microbatch(const bs_assign_t* a, int32_t k) {
  return (a && k >= 0 && k < (int32_t)a->mbs.size()) ? &a->mbs[k] : nullptr;
}
void bs_assign_destroy(bs_assign_t* a) { delete a; }

}  // extern "C"
