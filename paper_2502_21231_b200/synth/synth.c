/* synth.c — seeded, counter-based synthetic input generator (host only).
 *
 * Serves BOTH the oracle side and the CUDA side of the tests and bench.py, and therefore holds
 * none of the method's arithmetic: only pseudo-random numbers.  Counter-based so that any row of
 * any tensor can be regenerated on its own (sampled-row oracles at the 2M-token size never
 * materialise more than they need), and so that every CP rank's view of a sequence is a slice of
 * the same global tensor.
 *
 * Recipe: key = mix(seed, stream, seq); element e of the
 * [positions][row_elems] tensor of sequence `seq` draws u1 = U(key, 2e), u2 = U(key, 2e+1) with
 * U = SplitMix64 finaliser of (key + counter * golden), top 53 bits mapped into (0,1);
 * z = sqrt(-2 ln u1) cos(2 pi u2) (Box-Muller, cosine branch only); bf16 by round-to-nearest-even.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

static inline uint64_t mix64(uint64_t z) {
  z ^= z >> 30; z *= 0xbf58476d1ce4e5b9ULL;
  z ^= z >> 27; z *= 0x94d049bb133111ebULL;
  z ^= z >> 31;
  return z;
}
static inline uint64_t make_key(uint64_t seed, uint64_t stream, uint64_t seq) {
  uint64_t k = mix64(seed + 0x9e3779b97f4a7c15ULL);
  k = mix64(k ^ (stream * 0xd1342543de82ef95ULL + 0x632be59bd9b4e019ULL));
  k = mix64(k ^ (seq * 0xa0761d6478bd642fULL + 0xe7037ed1a0b428dbULL));
  return k;
}
static inline double unit_open(uint64_t key, uint64_t counter) { /* in (0,1) */
  uint64_t r = mix64(key + counter * 0x9e3779b97f4a7c15ULL);
  return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}
static inline double normal_at(uint64_t key, uint64_t e) {
  const double u1 = unit_open(key, 2 * e), u2 = unit_open(key, 2 * e + 1);
  return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}
static inline uint16_t f32_to_bf16_rne(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  u += 0x7fffu + ((u >> 16) & 1u); /* finite inputs only */
  return (uint16_t)(u >> 16);
}

/* out[i] = uniform in (0,1), i in [0,count), counters start..start+count-1 */
void synth_uniform_f64(uint64_t seed, uint64_t stream, uint64_t seq, uint64_t start,
                       uint64_t count, double* out) {
  const uint64_t key = make_key(seed, stream, seq);
  for (uint64_t i = 0; i < count; ++i) out[i] = unit_open(key, start + i);
}
void synth_normal_f64(uint64_t seed, uint64_t stream, uint64_t seq, uint64_t start,
                      uint64_t count, double* out) {
  const uint64_t key = make_key(seed, stream, seq);
  for (uint64_t i = 0; i < count; ++i) out[i] = normal_at(key, start + i);
}
/* Rows [pos_begin, pos_begin + n_rows) of the N(0,1) bf16 tensor [*][row_elems] of (seed,
 * stream, seq), written contiguously to out (n_rows * row_elems uint16). */
void synth_rows_bf16(uint64_t seed, uint64_t stream, uint64_t seq, uint64_t pos_begin,
                     uint64_t n_rows, uint64_t row_elems, uint16_t* out) {
  const uint64_t key = make_key(seed, stream, seq);
  const uint64_t n = n_rows * row_elems, e0 = pos_begin * row_elems;
#pragma omp parallel for schedule(static)
  for (uint64_t i = 0; i < n; ++i) out[i] = f32_to_bf16_rne((float)normal_at(key, e0 + i));
}
