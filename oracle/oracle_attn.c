/* oracle_attn.c — TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU oracle of the hot path.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with the CUDA path (paper_2502_21231_b200/csrc) and neither
 * includes the other.
 *
 * What it computes is the PLAIN DEFINITION (no tiling, no online softmax, no chunking):
 * the CUDA path (flash attention + chunk-and-merge) "optimizes memory I/O and employs the tiling
 * technique ... while still maintaining O(S^2) time complexity", i.e. it is exact
 * attention, so the oracle is masked softmax attention written out:
 *
 *   visible(i,j) <=> seq(i) == seq(j) and pos_k(j) <= pos_q(i)
 *        packing: "a special segmented attention mask to ensure that each sequence is processed
 *        independently by self-attention"; causal LM; CP "shards QKV along the
 *        sequence dimension" and must reproduce the same attention, so rows carry
 *        their GLOBAL position in their sequence.
 *   GQA: query head h reads kv head g = h / (Hq/Hkv)
 *   s_ij = scale * sum_d Q[i,h,d] K[j,g,d]            (softmax attention, ref [40] PAPER.md:471)
 *   LSE[h,i] = m_i + ln sum_j exp(s_ij - m_i),  m_i = max_j s_ij   (-inf if no visible key)
 *   P_ij = exp(s_ij - LSE[h,i]);   O[i,h,:] = sum_j P_ij V[j,g,:]  (0 if no visible key)
 *   delta_i = sum_d dO[i,h,d] O[i,h,d]
 *   dV[j,g,:] += P_ij dO[i,h,:];  dP_ij = sum_d dO[i,h,d] V[j,g,d];  dS_ij = P_ij (dP_ij - delta_i)
 *   dQ[i,h,:] += scale dS_ij K[j,g,:];   dK[j,g,:] += scale dS_ij Q[i,h,:]
 *   (gradients of softmax attention; flash-attention backward [7] PAPER.md:434 states the same)
 *
 * Inputs are bf16 bit patterns (uint16), converted EXACTLY to fp64.  All arithmetic is fp64.
 * Pins (tests/test_oracle_*.py): brute-force dense masked softmax in numpy, closed forms
 * (length-1 document, row 0, constant V, Q = 0), packing-order and chunk-and-merge invariance,
 * central finite differences, the gradient sum identities.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static inline double bf16_to_f64(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, 4);
  return (double)f;
}

int oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static inline int visible(const int32_t* q_seq, const int32_t* q_pos, const int32_t* k_seq,
                          const int32_t* k_pos, int64_t i, int64_t j) {
  return q_seq[i] == k_seq[j] && k_pos[j] <= q_pos[i];
}

/* s[j] for all visible j of row (h,i); returns number of visible keys; m = max. */
static int64_t scores_row(int64_t nk, int Hq, int Hkv, int D, const uint16_t* Q, const uint16_t* K,
                          const int32_t* q_seq, const int32_t* q_pos, const int32_t* k_seq,
                          const int32_t* k_pos, double scale, int h, int64_t i, double* s,
                          double* m_out) {
  const int g = h / (Hq / Hkv);
  const uint16_t* q = Q + ((size_t)i * Hq + h) * D;
  double m = -INFINITY;
  int64_t cnt = 0;
  for (int64_t j = 0; j < nk; ++j) {
    if (!visible(q_seq, q_pos, k_seq, k_pos, i, j)) {
      s[j] = -INFINITY;
      continue;
    }
    const uint16_t* k = K + ((size_t)j * Hkv + g) * D;
    double acc = 0.0;
    for (int d = 0; d < D; ++d) acc += bf16_to_f64(q[d]) * bf16_to_f64(k[d]);
    s[j] = scale * acc;
    if (s[j] > m) m = s[j];
    ++cnt;
  }
  *m_out = m;
  return cnt;
}

/* O: [nq,Hq,D] f64, LSE: [Hq,nq] f64.  Returns 0, or -1 on allocation failure. */
int oracle_attn_fwd(int64_t nq, int64_t nk, int Hq, int Hkv, int D, const uint16_t* Q,
                    const uint16_t* K, const uint16_t* V, const int32_t* q_seq,
                    const int32_t* q_pos, const int32_t* k_seq, const int32_t* k_pos, double scale,
                    double* O, double* LSE) {
  int fail = 0;
#pragma omp parallel
  {
    double* s = (double*)malloc(sizeof(double) * (size_t)(nk > 0 ? nk : 1));
    if (!s) {
#pragma omp atomic write
      fail = 1;
    }
#pragma omp barrier
    if (!fail) {
#pragma omp for collapse(2) schedule(dynamic, 16)
      for (int h = 0; h < Hq; ++h) {
        for (int64_t i = 0; i < nq; ++i) {
          const int g = h / (Hq / Hkv);
          double m;
          int64_t cnt = scores_row(nk, Hq, Hkv, D, Q, K, q_seq, q_pos, k_seq, k_pos, scale, h, i,
                                   s, &m);
          double* o = O + ((size_t)i * Hq + h) * D;
          for (int d = 0; d < D; ++d) o[d] = 0.0;
          if (cnt == 0) {
            LSE[(size_t)h * nq + i] = -INFINITY;
            continue;
          }
          double l = 0.0;
          for (int64_t j = 0; j < nk; ++j)
            if (s[j] != -INFINITY) l += exp(s[j] - m);
          const double lse = m + log(l);
          LSE[(size_t)h * nq + i] = lse;
          for (int64_t j = 0; j < nk; ++j) {
            if (s[j] == -INFINITY) continue;
            const double p = exp(s[j] - lse);
            const uint16_t* v = V + ((size_t)j * Hkv + g) * D;
            for (int d = 0; d < D; ++d) o[d] += p * bf16_to_f64(v[d]);
          }
        }
      }
    }
    free(s);
  }
  return fail ? -1 : 0;
}

/* Gradients.  dQ: [nq,Hq,D], dK,dV: [nk,Hkv,D] f64, all OVERWRITTEN.
 * LSE_in / delta_in ([Hq,nq] f64) may be NULL: then LSE and delta are those of THIS key set
 * (the plain definition).  When given (the merged LSE and delta of a larger key set), the
 * result is this key set's exact share of the gradients of attention over the larger set
 * (reading 13; the sum over a partition of the keys equals the full backward, which
 * tests/test_oracle_attn.py checks).
 * Written as the formulas read: pass A, one query row (h,i) at a time: LSE_i, delta_i and
 * dQ[i,h,:] = scale sum_j dS_ij K[j,g,:];  pass B, one key row (g,j) at a time:
 * dV[j,g,:] = sum_{h in g} sum_i P_ij dO[i,h,:] and dK[j,g,:] = scale sum_{h in g} sum_i dS_ij
 * Q[i,h,:].  Each output row is owned by one loop iteration, so the loops parallelise as is. */
int oracle_attn_bwd(int64_t nq, int64_t nk, int Hq, int Hkv, int D, const uint16_t* Q,
                    const uint16_t* K, const uint16_t* V, const uint16_t* dO, const int32_t* q_seq,
                    const int32_t* q_pos, const int32_t* k_seq, const int32_t* k_pos, double scale,
                    const double* LSE_in, const double* delta_in, double* dQ, double* dK,
                    double* dV) {
  int fail = 0;
  const int G = Hq / Hkv;
  double* LSE = (double*)malloc(sizeof(double) * (size_t)(nq * Hq > 0 ? nq * Hq : 1));
  double* delta = (double*)malloc(sizeof(double) * (size_t)(nq * Hq > 0 ? nq * Hq : 1));
  if (!LSE || !delta) {
    free(LSE);
    free(delta);
    return -1;
  }
  memset(dQ, 0, sizeof(double) * (size_t)nq * Hq * D);
  memset(dK, 0, sizeof(double) * (size_t)nk * Hkv * D);
  memset(dV, 0, sizeof(double) * (size_t)nk * Hkv * D);
#pragma omp parallel
  {
    double* s = (double*)malloc(sizeof(double) * (size_t)(nk > 0 ? nk : 1));
    double* o = (double*)malloc(sizeof(double) * (size_t)D);
    if (!s || !o) {
#pragma omp atomic write
      fail = 1;
    }
#pragma omp barrier
    if (!fail) {
      /* pass A: per query row */
#pragma omp for collapse(2) schedule(dynamic, 16)
      for (int h = 0; h < Hq; ++h) {
        for (int64_t i = 0; i < nq; ++i) {
          const int g = h / G;
          double m;
          int64_t cnt =
              scores_row(nk, Hq, Hkv, D, Q, K, q_seq, q_pos, k_seq, k_pos, scale, h, i, s, &m);
          double lse = -INFINITY, dl = 0.0;
          const uint16_t* go = dO + ((size_t)i * Hq + h) * D;
          if (cnt > 0) {
            if (LSE_in) {
              lse = LSE_in[(size_t)h * nq + i];
              dl = delta_in[(size_t)h * nq + i];
            } else {
              double l = 0.0;
              for (int64_t j = 0; j < nk; ++j)
                if (s[j] != -INFINITY) l += exp(s[j] - m);
              lse = m + log(l);
              for (int d = 0; d < D; ++d) o[d] = 0.0;
              for (int64_t j = 0; j < nk; ++j) {
                if (s[j] == -INFINITY) continue;
                const double p = exp(s[j] - lse);
                const uint16_t* v = V + ((size_t)j * Hkv + g) * D;
                for (int d = 0; d < D; ++d) o[d] += p * bf16_to_f64(v[d]);
              }
              for (int d = 0; d < D; ++d) dl += bf16_to_f64(go[d]) * o[d];
            }
            double* dq = dQ + ((size_t)i * Hq + h) * D;
            for (int64_t j = 0; j < nk; ++j) {
              if (s[j] == -INFINITY) continue;
              const double p = exp(s[j] - lse);
              const uint16_t* k = K + ((size_t)j * Hkv + g) * D;
              const uint16_t* v = V + ((size_t)j * Hkv + g) * D;
              double dp = 0.0;
              for (int d = 0; d < D; ++d) dp += bf16_to_f64(go[d]) * bf16_to_f64(v[d]);
              const double ds = p * (dp - dl);
              for (int d = 0; d < D; ++d) dq[d] += scale * ds * bf16_to_f64(k[d]);
            }
          }
          LSE[(size_t)h * nq + i] = lse;
          delta[(size_t)h * nq + i] = dl;
        }
      }
      /* pass B: per key row (implicit barrier of the omp-for above orders the two passes) */
#pragma omp for collapse(2) schedule(dynamic, 16)
      for (int g = 0; g < Hkv; ++g) {
        for (int64_t j = 0; j < nk; ++j) {
          const uint16_t* k = K + ((size_t)j * Hkv + g) * D;
          const uint16_t* v = V + ((size_t)j * Hkv + g) * D;
          double* dk = dK + ((size_t)j * Hkv + g) * D;
          double* dv = dV + ((size_t)j * Hkv + g) * D;
          for (int h = g * G; h < (g + 1) * G; ++h) {
            for (int64_t i = 0; i < nq; ++i) {
              if (!visible(q_seq, q_pos, k_seq, k_pos, i, j)) continue;
              const uint16_t* q = Q + ((size_t)i * Hq + h) * D;
              const uint16_t* go = dO + ((size_t)i * Hq + h) * D;
              double acc = 0.0, dp = 0.0;
              for (int d = 0; d < D; ++d) {
                acc += bf16_to_f64(q[d]) * bf16_to_f64(k[d]);
                dp += bf16_to_f64(go[d]) * bf16_to_f64(v[d]);
              }
              const double p = exp(scale * acc - LSE[(size_t)h * nq + i]);
              const double ds = p * (dp - delta[(size_t)h * nq + i]);
              for (int d = 0; d < D; ++d) {
                dv[d] += p * bf16_to_f64(go[d]);
                dk[d] += scale * ds * bf16_to_f64(q[d]);
              }
            }
          }
        }
      }
    }
    free(s);
    free(o);
  }
  free(LSE);
  free(delta);
  return fail ? -1 : 0;
}

/* LSE merge of n partials (BASELINE.json north_star: "a separate merge combines the partials";
 * ring attention [25] PAPER.md:454; reading 2):
 *   M = max_s LSE_s; if M == -inf: LSE = -inf, O = 0
 *   else w_s = exp(LSE_s - M), Z = sum_s w_s, LSE = M + ln Z, O = sum_s (w_s / Z) O_s
 * O_parts: [n][rows,Hq,D] f64 contiguous; LSE_parts: [n][Hq,rows] f64 contiguous. */
int oracle_merge(int n, int64_t rows, int Hq, int D, const double* O_parts,
                 const double* LSE_parts, double* O, double* LSE) {
  const size_t o_sz = (size_t)rows * Hq * D, l_sz = (size_t)rows * Hq;
#pragma omp parallel for collapse(2)
  for (int h = 0; h < Hq; ++h) {
    for (int64_t i = 0; i < rows; ++i) {
      double M = -INFINITY;
      for (int s = 0; s < n; ++s) {
        const double v = LSE_parts[s * l_sz + (size_t)h * rows + i];
        if (v > M) M = v;
      }
      double* o = O + ((size_t)i * Hq + h) * D;
      for (int d = 0; d < D; ++d) o[d] = 0.0;
      if (M == -INFINITY) {
        LSE[(size_t)h * rows + i] = -INFINITY;
        continue;
      }
      double Z = 0.0;
      for (int s = 0; s < n; ++s) Z += exp(LSE_parts[s * l_sz + (size_t)h * rows + i] - M);
      LSE[(size_t)h * rows + i] = M + log(Z);
      for (int s = 0; s < n; ++s) {
        const double w = exp(LSE_parts[s * l_sz + (size_t)h * rows + i] - M) / Z;
        if (w == 0.0) continue; /* a part with LSE = -inf carries no weight (and may hold anything) */
        const double* os = O_parts + s * o_sz + ((size_t)i * Hq + h) * D;
        for (int d = 0; d < D; ++d) o[d] += w * os[d];
      }
    }
  }
  return 0;
}
