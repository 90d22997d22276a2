// assign.cpp — bs_assign: the naive HDP solution (Algorithm 1; routine at
// PAPER.md:262) with offload ratio r = 0, host integers only.  The step directly upstream of
// bs_plan: a global batch of sequence lengths becomes, for every HDP rank and every round of the
// step, the bs_seq_t list that rank hands to bs_plan.  Readings R1-R4: include/bytescale_attn.h.
// bs_balance: the balance strategy (Algorithm 2, DP-Balance) over the same groups, readings B1-B6.
#include <algorithm>
#include <map>
#include <new>
#include <vector>

#include "common.h"

struct bs_balance_s {
  std::vector<int64_t> exec_times;
  int64_t makespan = 0;
  std::vector<bs_seq_t> seqs;
  std::vector<int32_t> src;
  std::vector<bs_timed_microbatch_t> mbs;  // sorted by (rank, start)
};

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

// Lines 1-9 of Algorithm 1, shared by bs_assign and bs_balance: D(s_i), then the groups - the long
// sequences in input order (one entry {len, cp = D, 0} each), then the bins of whole sequences.
struct Groups {
  std::vector<int32_t> d;
  std::vector<bs_seq_t> seqs;
  std::vector<int32_t> src;
  std::vector<Pending> groups;
};

bs_status_t make_groups(const char* who, const int32_t* lens, int32_t n, int32_t capacity,
                        int32_t d_hdp, Groups* out) {
  BS_REQUIRE(n >= 0 && (lens != nullptr || n == 0), BS_ERR_INVALID_ARG, "%s: bad lens / n", who);
  BS_REQUIRE(capacity >= 1 && d_hdp >= 1, BS_ERR_INVALID_ARG,
             "%s: capacity %d and d_hdp %d must be positive", who, capacity, d_hdp);
  out->d.resize(n);
  // lines 1-6: D(s_i) = ceil(s_i / C) (Eq. 3 with r = 0, Act linear); D = 1 goes to the pack list
  std::multimap<int32_t, int32_t, std::greater<int32_t>> pack;  // length (descending) -> index
  std::vector<int32_t> longs;
  for (int32_t i = 0; i < n; ++i) {
    BS_REQUIRE(lens[i] >= 1, BS_ERR_INVALID_ARG, "%s: sequence %d has length %d", who, i, lens[i]);
    const int64_t d = ((int64_t)lens[i] + capacity - 1) / capacity;
    BS_REQUIRE(d <= d_hdp, BS_ERR_INVALID_ARG,
               "%s: sequence %d (%d tokens) needs %lld ranks of capacity %d, d_hdp is %d", who, i,
               lens[i], (long long)d, capacity, d_hdp);
    out->d[i] = (int32_t)d;
    if (d == 1)
      pack.emplace(lens[i], i);  // equal lengths keep input order (multimap insertion order)
    else
      longs.push_back(i);
  }
  // long sequences first, in input order
  for (int32_t i : longs) {
    const int32_t b = (int32_t)out->seqs.size();
    out->seqs.push_back({lens[i], out->d[i], 0});
    out->src.push_back(i);
    out->groups.push_back({out->d[i], b, b + 1, 0, 0});
  }
  // lines 7-9: one bin per pass; the longest remaining sequence that still fits, until none does
  while (!pack.empty()) {
    int32_t room = capacity;
    const int32_t b = (int32_t)out->seqs.size();
    for (;;) {
      auto it = pack.lower_bound(room);  // first key <= room in descending order
      if (it == pack.end()) break;
      room -= it->first;
      out->seqs.push_back({it->first, 1, 0});
      out->src.push_back(it->second);
      pack.erase(it);
    }
    out->groups.push_back({1, b, (int32_t)out->seqs.size(), 0, 0});
  }
  return BS_OK;
}

}  // namespace

extern "C" {

bs_status_t bs_assign(const int32_t* lens, int32_t n, int32_t capacity, int32_t d_hdp,
                      bs_assign_t** out) {
  BS_REQUIRE(out != nullptr, BS_ERR_INVALID_ARG, "bs_assign: out is null");
  *out = nullptr;
  try {
    Groups gr;
    bs_status_t rc = make_groups("bs_assign", lens, n, capacity, d_hdp, &gr);
    if (rc != BS_OK) return rc;
    bs_assign_s* a = new bs_assign_s;
    struct Guard {
      bs_assign_s* p;
      ~Guard() { delete p; }
    } guard{a};
    a->d.swap(gr.d);
    a->seqs.swap(gr.seqs);
    a->src.swap(gr.src);
    std::vector<Pending>& groups = gr.groups;
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

// bs_balance: Algorithm 2, DP-Balance, in place of line 10 of Algorithm 1.
bs_status_t bs_balance(const int32_t* lens, int32_t n, int32_t capacity, int32_t d_hdp,
                       const int64_t* cost, int32_t n_buckets, int64_t delta, bs_balance_t** out) {
  BS_REQUIRE(out != nullptr, BS_ERR_INVALID_ARG, "bs_balance: out is null");
  *out = nullptr;
  BS_REQUIRE(cost != nullptr && cost[0] >= 0 && cost[1] >= 0 && cost[2] >= 0, BS_ERR_INVALID_ARG,
             "bs_balance: cost coefficients must be three non-negative integers");
  BS_REQUIRE(n_buckets >= 1 && delta >= 0, BS_ERR_INVALID_ARG,
             "bs_balance: n_buckets %d must be positive, delta %lld non-negative", n_buckets,
             (long long)delta);
  try {
    Groups gr;
    bs_status_t rc = make_groups("bs_balance", lens, n, capacity, d_hdp, &gr);
    if (rc != BS_OK) return rc;
    // B1: time a group costs each of its ranks
    const int64_t kLimit = (int64_t)1 << 53;
    auto seq_time = [&](int64_t s, int64_t* t) -> bool {
      const __int128 v = (__int128)cost[0] * s * s + (__int128)cost[1] * s + cost[2];
      *t = (int64_t)v;
      return v < kLimit;
    };
    struct Job {
      int64_t time;
      int32_t ranks, group;
    };
    std::vector<Job> jobs;
    __int128 total = 0;
    for (size_t g = 0; g < gr.groups.size(); ++g) {
      const Pending& p = gr.groups[g];
      int64_t time = 0;
      for (int32_t q = p.seq_begin; q < p.seq_end; ++q) {
        int64_t t;
        BS_REQUIRE(seq_time(gr.seqs[q].len, &t) && time + t < kLimit, BS_ERR_INVALID_ARG,
                   "bs_balance: the cost of sequence %d does not fit 2^53", gr.src[q]);
        time += t;
      }
      if (p.ranks > 1) time /= p.ranks;
      jobs.push_back({time, p.ranks, (int32_t)g});
      total += (__int128)time * p.ranks;
    }
    BS_REQUIRE(total < ((__int128)1 << 62), BS_ERR_INVALID_ARG, "bs_balance: total cost overflows");
    // lines 3-5 (B2, B3): longest first.  Under DP-Balance the groups leave the buckets in exactly
    // this order (first bucket first, B6), so the bucket boundaries need not be materialised.
    std::stable_sort(jobs.begin(), jobs.end(), [](const Job& x, const Job& y) {
      return x.time != y.time ? x.time > y.time : x.ranks > y.ranks;
    });
    bs_balance_s* b = new bs_balance_s;
    struct Guard {
      bs_balance_s* p;
      ~Guard() { delete p; }
    } guard{b};
    b->exec_times.assign(d_hdp, 0);
    struct Slot {
      int32_t rank;
      int64_t start, end;
      int32_t begin, count;
    };
    std::vector<Slot> slots;
    std::vector<int32_t> by_load(d_hdp);
    for (const Job& job : jobs) {
      // lines 7-17 (B4, B5): the ranks that lag more than delta behind the slowest one are the
      // least loaded ones, and when fewer than D lag the least loaded others fill up - either way
      // the group goes to the D least loaded ranks (ties: lowest rank), which start together.
      for (int32_t i = 0; i < d_hdp; ++i) by_load[i] = i;
      std::partial_sort(by_load.begin(), by_load.begin() + job.ranks, by_load.end(),
                        [&](int32_t x, int32_t y) {
                          return b->exec_times[x] != b->exec_times[y]
                                     ? b->exec_times[x] < b->exec_times[y] : x < y;
                        });
      std::sort(by_load.begin(), by_load.begin() + job.ranks);
      int64_t start = 0;
      for (int32_t j = 0; j < job.ranks; ++j) start = std::max(start, b->exec_times[by_load[j]]);
      const int64_t end = start + job.time;
      const Pending& p = gr.groups[job.group];
      for (int32_t j = 0; j < job.ranks; ++j) {
        b->exec_times[by_load[j]] = end;
        const int32_t at = (int32_t)b->seqs.size();
        if (job.ranks > 1) {
          bs_seq_t s = gr.seqs[p.seq_begin];
          s.rank = j;
          b->seqs.push_back(s);
          b->src.push_back(gr.src[p.seq_begin]);
        } else {
          b->seqs.insert(b->seqs.end(), gr.seqs.begin() + p.seq_begin, gr.seqs.begin() + p.seq_end);
          b->src.insert(b->src.end(), gr.src.begin() + p.seq_begin, gr.src.begin() + p.seq_end);
        }
        slots.push_back({by_load[j], start, end, at, (int32_t)b->seqs.size() - at});
      }
    }
    for (int64_t t : b->exec_times) b->makespan = std::max(b->makespan, t);
    std::stable_sort(slots.begin(), slots.end(), [](const Slot& x, const Slot& y) {
      return x.rank != y.rank ? x.rank < y.rank : x.start < y.start;
    });
    for (const Slot& s : slots)
      b->mbs.push_back({s.rank, s.count, s.start, s.end, b->seqs.data() + s.begin,
                        b->src.data() + s.begin});
    guard.p = nullptr;
    *out = b;
    return BS_OK;
  } catch (const std::bad_alloc&) {
    return bs::fail(BS_ERR_HOST_OOM, "bs_balance: out of host memory");
  }
}

int32_t bs_balance_n_ranks(const bs_balance_t* b) { return b ? (int32_t)b->exec_times.size() : 0; }
const int64_t* bs_balance_exec_times(const bs_balance_t* b) {
  return b ? b->exec_times.data() : nullptr;
}
int64_t bs_balance_makespan(const bs_balance_t* b) { return b ? b->makespan : 0; }
int32_t bs_balance_n_microbatches(const bs_balance_t* b) { return b ? (int32_t)b->mbs.size() : 0; }
const bs_timed_microbatch_t* bs_balance_microbatch(const bs_balance_t* b, int32_t k) {
  return (b && k >= 0 && k < (int32_t)b->mbs.size()) ? &b->mbs[k] : nullptr;
}
void bs_balance_destroy(bs_balance_t* b) { delete b; }

}  // extern "C"
