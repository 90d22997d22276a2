// plan.cpp — bs_plan: data-aware sharding, device-local view (host, integers only).
//
// "each sequence is processed by the minimal number of ranks": a sequence with
// cp == 1 stays whole; one with cp == N is cut into 2N parts, rank r holding parts r and 2N-1-r
// so every rank owns 1/N of the tokens and 1/N of the causal mask area; KV chunks
// arrive in ring order.  Canonical form: include/bytescale_attn.h.
#include <new>
#include <vector>

#include "common.h"

struct bs_plan_s {
  struct Step {
    std::vector<bs_seg_t> segs;
    std::vector<int32_t> kv_seq, kv_src_rank, cu_rows_k, k_pos, k_seq;
    bs_step_t pub;
  };
  int32_t n_seqs = 0;
  std::vector<int32_t> cu_rows_q, q_pos, q_seq;
  std::vector<Step> steps;
};

namespace {

struct Part {
  int64_t begin, len;  // global start position, token count
};

// Part k of a sequence split 2N ways: [floor(k*len/2N), floor((k+1)*len/2N)).
inline Part part_of(int64_t len, int64_t cp, int64_t k) {
  const int64_t b = (k * len) / (2 * cp), e = ((k + 1) * len) / (2 * cp);
  return {b, e - b};
}
// (low, high) parts held by rank p; high is empty for cp == 1.
inline void held(const bs_seq_t& s, int32_t p, Part out[2]) {
  if (s.cp == 1) {
    out[0] = {0, s.len};
    out[1] = {0, 0};
  } else {
    out[0] = part_of(s.len, s.cp, p);
    out[1] = part_of(s.len, s.cp, 2 * (int64_t)s.cp - 1 - p);
  }
}
// sum_{a=0}^{q_len-1} clamp(a + off + 1, 0, k_len), closed form.
inline int64_t visible_pairs(int64_t q_len, int64_t k_len, int64_t off) {
  int64_t a0 = off < 0 ? -off : 0;  // first row that sees key 0
  if (a0 >= q_len) return 0;
  int64_t a1 = k_len - off - 1;  // first row that sees every key
  if (a1 < a0) a1 = a0;
  if (a1 > q_len) a1 = q_len;
  const int64_t n = a1 - a0;
  return n * (off + 1) + (a0 + a1 - 1) * n / 2 + (q_len - a1) * k_len;
}

}  // namespace

extern "C" {

bs_status_t bs_plan(const bs_seq_t* seqs, int32_t n_seqs, bs_plan_t** out) {
  BS_REQUIRE(out != nullptr, BS_ERR_INVALID_ARG, "bs_plan: out is null");
  *out = nullptr;
  BS_REQUIRE(n_seqs >= 0, BS_ERR_INVALID_ARG, "bs_plan: n_seqs = %d < 0", n_seqs);
  BS_REQUIRE(seqs != nullptr || n_seqs == 0, BS_ERR_INVALID_ARG, "bs_plan: seqs is null");
  int32_t max_cp = 0;
  int64_t total = 0;
  for (int32_t i = 0; i < n_seqs; ++i) {
    const bs_seq_t& s = seqs[i];
    BS_REQUIRE(s.len >= 1, BS_ERR_INVALID_ARG, "bs_plan: seqs[%d].len = %d < 1", i, s.len);
    BS_REQUIRE(s.cp >= 1, BS_ERR_INVALID_ARG, "bs_plan: seqs[%d].cp = %d < 1", i, s.cp);
    BS_REQUIRE(s.rank >= 0 && s.rank < s.cp, BS_ERR_INVALID_ARG,
               "bs_plan: seqs[%d].rank = %d outside [0,%d)", i, s.rank, s.cp);
    if (s.cp > max_cp) max_cp = s.cp;
    Part h[2];
    held(s, s.rank, h);
    total += h[0].len + h[1].len;
    // any rank's chunk can be this device's KV buffer: bound the largest one too
    BS_REQUIRE(total <= INT32_MAX - 4 * (int64_t)n_seqs, BS_ERR_INVALID_ARG,
               "bs_plan: more than INT32_MAX local rows");
  }
  bs_plan_s* p = nullptr;
  try {
    p = new bs_plan_s();
    p->n_seqs = n_seqs;
    p->cu_rows_q.assign(1, 0);
    std::vector<Part> qparts(2 * (size_t)n_seqs);
    std::vector<int32_t> qrow(2 * (size_t)n_seqs);
    for (int32_t i = 0; i < n_seqs; ++i) {
      held(seqs[i], seqs[i].rank, &qparts[2 * i]);
      int32_t row = p->cu_rows_q.back();
      for (int t = 0; t < 2; ++t) {
        qrow[2 * i + t] = row;
        for (int64_t a = 0; a < qparts[2 * i + t].len; ++a) {
          p->q_pos.push_back((int32_t)(qparts[2 * i + t].begin + a));
          p->q_seq.push_back(i);
        }
        row += (int32_t)qparts[2 * i + t].len;
      }
      p->cu_rows_q.push_back(row);
    }
    p->steps.resize(max_cp);
    for (int32_t s = 0; s < max_cp; ++s) {
      bs_plan_s::Step& st = p->steps[s];
      st.cu_rows_k.assign(1, 0);
      int64_t pairs = 0;
      for (int32_t i = 0; i < n_seqs; ++i) {
        const bs_seq_t& sq = seqs[i];
        if (sq.cp <= s) continue;
        const int32_t src = ((sq.rank - s) % sq.cp + sq.cp) % sq.cp;
        Part kp[2];
        held(sq, src, kp);
        int32_t krow[2];
        int32_t row = st.cu_rows_k.back();
        for (int t = 0; t < 2; ++t) {
          krow[t] = row;
          for (int64_t b = 0; b < kp[t].len; ++b) {
            st.k_pos.push_back((int32_t)(kp[t].begin + b));
            st.k_seq.push_back(i);
          }
          row += (int32_t)kp[t].len;
        }
        st.kv_seq.push_back(i);
        st.kv_src_rank.push_back(src);
        st.cu_rows_k.push_back(row);
        for (int tq = 0; tq < 2; ++tq) {
          const Part& q = qparts[2 * i + tq];
          for (int tk = 0; tk < 2; ++tk) {
            const Part& k = kp[tk];
            if (q.len == 0 || k.len == 0) continue;
            if (k.begin > q.begin + q.len - 1) continue;  // no visible pair
            bs_seg_t g;
            g.q_begin = qrow[2 * i + tq];
            g.q_end = g.q_begin + (int32_t)q.len;
            g.k_begin = krow[tk];
            g.k_end = g.k_begin + (int32_t)k.len;
            g.causal_offset = (int32_t)(q.begin - k.begin);
            g.seq = i;
            st.segs.push_back(g);
            pairs += visible_pairs(q.len, k.len, q.begin - k.begin);
          }
        }
      }
      st.pub.step = s;
      st.pub.n_segs = (int32_t)st.segs.size();
      st.pub.segs = st.segs.data();
      st.pub.kv_rows = st.cu_rows_k.back();
      st.pub.n_kv_seqs = (int32_t)st.kv_seq.size();
      st.pub.kv_seq = st.kv_seq.data();
      st.pub.kv_src_rank = st.kv_src_rank.data();
      st.pub.cu_rows_k = st.cu_rows_k.data();
      st.pub.visible_pairs = pairs;
    }
  } catch (const std::bad_alloc&) {
    delete p;
    return bs::fail(BS_ERR_HOST_OOM, "bs_plan: out of host memory");
  }
  *out = p;
  return BS_OK;
}

bs_status_t bs_plan_uniform(const int32_t* lens, int32_t n, int32_t cp, int32_t rank,
                            int32_t min_shard_len, bs_plan_t** out) {
  BS_REQUIRE(out != nullptr, BS_ERR_INVALID_ARG, "bs_plan_uniform: out is null");
  *out = nullptr;
  BS_REQUIRE(n >= 0 && (lens != nullptr || n == 0), BS_ERR_INVALID_ARG,
             "bs_plan_uniform: bad lens/n");
  BS_REQUIRE(cp >= 1 && rank >= 0 && rank < cp, BS_ERR_INVALID_ARG,
             "bs_plan_uniform: rank %d outside [0,%d)", rank, cp);
  std::vector<bs_seq_t> seqs;
  try {
    seqs.resize((size_t)n);
  } catch (const std::bad_alloc&) {
    return bs::fail(BS_ERR_HOST_OOM, "bs_plan_uniform: out of host memory");
  }
  for (int32_t i = 0; i < n; ++i) {
    const bool shard = cp > 1 && lens[i] >= min_shard_len;
    seqs[i] = {lens[i], shard ? cp : 1, shard ? rank : 0};
  }
  return bs_plan(seqs.data(), n, out);
}

int32_t bs_plan_n_seqs(const bs_plan_t* p) { return p ? p->n_seqs : 0; }
int32_t bs_plan_q_rows(const bs_plan_t* p) { return p ? p->cu_rows_q.back() : 0; }
const int32_t* bs_plan_cu_rows_q(const bs_plan_t* p) { return p ? p->cu_rows_q.data() : nullptr; }
const int32_t* bs_plan_q_pos(const bs_plan_t* p) { return p ? p->q_pos.data() : nullptr; }
const int32_t* bs_plan_q_seq(const bs_plan_t* p) { return p ? p->q_seq.data() : nullptr; }
int32_t bs_plan_n_steps(const bs_plan_t* p) { return p ? (int32_t)p->steps.size() : 0; }
const bs_step_t* bs_plan_step(const bs_plan_t* p, int32_t s) {
  if (!p || s < 0 || s >= (int32_t)p->steps.size()) return nullptr;
  return &p->steps[s].pub;
}
const int32_t* bs_plan_step_k_pos(const bs_plan_t* p, int32_t s) {
  if (!p || s < 0 || s >= (int32_t)p->steps.size()) return nullptr;
  return p->steps[s].k_pos.data();
}
const int32_t* bs_plan_step_k_seq(const bs_plan_t* p, int32_t s) {
  if (!p || s < 0 || s >= (int32_t)p->steps.size()) return nullptr;
  return p->steps[s].k_seq.data();
}
void bs_plan_destroy(bs_plan_t* p) { delete p; }

}  // extern "C"
