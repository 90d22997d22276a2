/* bytescale_attn.h — C-ABI boundary of the B200-native ByteScale attention hot path.
 *
 * What this library is: the per-device data-parallel hot path of one Hybrid Data Parallelism
 * (HDP) rank of ByteScale (arXiv 2502.21231; PAPER.md = /root/reference/PAPER.md):
 * causal self-attention over a packed buffer of variable-length documents ("packing ... employs
 * a special segmented attention mask to ensure that each sequence is processed independently",
 * PAPER.md:93) in which some sequences are whole and others are zigzag context-parallel shards
 * ("each subsequence ... is uniformly divided into 2N parts and symmetrically assigned to the N
 * devices"), computed one Q-chunk x KV-chunk ring step at a time,
 * each step returning a partial O and a per-row natural-log LSE; a separate LSE merge; and the
 * matching backward.  BASELINE.json north_star fixes the call list.
 *
 * Conventions for every entry point
 *   - extern "C"; plain pointers and sizes; no exception crosses the boundary; nothing prints.
 *   - Every function returning bs_status_t returns BS_OK (0) or a negative code; the detail text
 *     is available from bs_last_error() (thread-local, valid until the next call on the thread).
 *   - "device" pointers are CUDA device memory owned by the caller; "host" pointers are ordinary
 *     host memory.  The library never allocates or frees device memory, and never synchronises
 *     the device: all device work is enqueued on `stream` (a cudaStream_t passed as void*; NULL =
 *     the legacy default stream).  Host arrays may be freed as soon as the call returns.
 *     bs_attn_fwd / bs_attn_bwd stage their work-item tables in pinned host memory owned by the
 *     library (a ring of 64 slots, allocated on first use, never freed) and copy them with one
 *     DMA on `stream`; the host waits only when 64 such copies are still in flight.  Because the
 *     slots are reused, these two calls must not be captured into a CUDA graph.
 *   - Every argument check (shapes, ranges, segment consistency, workspace, alignment of every
 *     pointer and stride, the device) is made before anything is enqueued: a call that returns
 *     an error has written nothing.
 *   - Rows of the buffers that no segment of a call references may hold anything, NaN and Inf
 *     included (fixed-capacity or uninitialised padding): they never reach a result.
 *   - Tensors: Q, O, dO, dQ are [q_rows][n_q_heads][head_dim] bf16 with dim stride 1, head stride
 *     head_dim and row stride q_row_stride elements.  K, V, dK, dV are
 *     [kv_rows][n_kv_heads][head_dim] bf16 with row stride kv_row_stride.  LSE and delta are fp32,
 *     element (h, row) at [h * lse_head_stride + row].  dQ_acc is fp32 [q_rows][n_q_heads][head_dim]
 *     densely packed.  Base pointers must be 16-byte aligned, row strides multiples of 8 elements.
 *   - head_dim in {64, 128}; n_q_heads % n_kv_heads == 0 (GQA).
 */
#ifndef BYTESCALE_ATTN_H_
#define BYTESCALE_ATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BS_VERSION 100 /* 0.1.0 */

typedef enum {
  BS_OK = 0,
  BS_ERR_INVALID_ARG = -1, /* null pointer, bad range, bad stride, inconsistent segments */
  BS_ERR_UNSUPPORTED = -2, /* head_dim not in {64,128}; more than 2^30 - 1024 rows in a buffer; the
                              current device is not compute capability 10.0 (checked by every
                              device call before anything is enqueued) */
  BS_ERR_WORKSPACE = -3,   /* workspace null / too small / misaligned */
  BS_ERR_CUDA = -4,        /* a CUDA runtime/driver call failed; text from cudaGetErrorString */
  BS_ERR_HOST_OOM = -5
} bs_status_t;

const char* bs_status_string(bs_status_t s); /* static storage */
const char* bs_last_error(void);             /* thread-local detail of the last failure */
int bs_version(void);

/* ------------------------------------------------------------------------------------------ */
/* Planning — host only, integers only.  Data-aware sharding, device-local view:               */
/* "each sequence is processed by the minimal number of ranks"; long sequences   */
/* are zigzag-split 2N ways, rank r holding parts r and 2N-1-r; KV chunks arrive  */
/* in ring order.  Canonical form:            */
/*   parts   : cp == 1 -> one part [0,len); cp == N >= 2 -> part k = [floor(k*len/2N),           */
/*             floor((k+1)*len/2N)), k in [0,2N); rank p holds part p ("low") and 2N-1-p ("high") */
/*   Q buffer: sequences in input order, low part rows then high part rows                      */
/*   steps   : n_steps = max cp; at step s the sequences with cp > s take part, source rank      */
/*             p = (rank - s) mod cp; the step's KV buffer = [low part of p ; high part of p]    */
/*             per participating sequence, in input order                                       */
/*   segments: per participating sequence, for q part in (low, high), for k part in (low, high): */
/*             emitted iff both parts are non-empty and at least one pair is visible;            */
/*             causal_offset = q_part_global_start - k_part_global_start (unclamped)             */
/* ------------------------------------------------------------------------------------------ */

typedef struct {
  int32_t len;  /* full sequence length in tokens, >= 1 */
  int32_t cp;   /* context-parallel degree N of this sequence; 1 = whole on this device */
  int32_t rank; /* this device's rank inside the sequence's CP group, 0 <= rank < cp */
} bs_seq_t;

/* One rectangular piece of attention work: queries = rows [q_begin,q_end) of the Q-side buffers,
 * keys = rows [k_begin,k_end) of THIS call's K/V buffers.  With a, b the 0-based indices inside
 * the two ranges, key b is visible to query a iff  b <= a + causal_offset.
 * Two segments of one call have identical or disjoint q ranges; a row's softmax runs over the
 * union of the visible keys of every segment that contains the row.  bs_attn_bwd additionally
 * needs the k ranges of two segments to be identical or disjoint (it owns dK / dV per key range;
 * bs_plan's segments satisfy both rules).  causal_offset may be any int32: offsets >= k_len - 1
 * mean "every key", offsets <= -q_len "no key" (INT32_MAX / INT32_MIN are fine); the library
 * clamps it to [-q_len, k_len], which leaves the mask unchanged. */
typedef struct {
  int32_t q_begin, q_end;
  int32_t k_begin, k_end;
  int32_t causal_offset;
  int32_t seq; /* index into the planner's input seqs[] (informational for device calls) */
} bs_seg_t;

typedef struct {
  int32_t step;               /* ring step index s */
  int32_t n_segs;
  const bs_seg_t* segs;       /* [n_segs], owned by the plan */
  int32_t kv_rows;            /* rows of this step's K/V buffer */
  int32_t n_kv_seqs;          /* sequences present in this step's K/V buffer */
  const int32_t* kv_seq;      /* [n_kv_seqs] sequence indices, input order */
  const int32_t* kv_src_rank; /* [n_kv_seqs] CP rank whose K/V this is: (rank - s) mod cp */
  const int32_t* cu_rows_k;   /* [n_kv_seqs + 1] first K/V row of each present sequence */
  int64_t visible_pairs;      /* visible (query,key) pairs of the step, per head */
} bs_step_t;

typedef struct bs_plan_s bs_plan_t; /* opaque, host memory owned by the library */

/* Build the plan for this device.  seqs: host, [n_seqs].  *out receives a plan to be released
 * with bs_plan_destroy.  Errors: INVALID_ARG (null, n_seqs < 0, len < 1, cp < 1, rank out of
 * range, total rows > INT32_MAX), HOST_OOM. */
bs_status_t bs_plan(const bs_seq_t* seqs, int32_t n_seqs, bs_plan_t** out);

/* Convenience form of north_star's "per-sequence lengths and a CP degree": sequences with
 * len >= min_shard_len get (cp, rank); all others cp = 1, rank = 0. */
bs_status_t bs_plan_uniform(const int32_t* lens, int32_t n, int32_t cp, int32_t rank,
                            int32_t min_shard_len, bs_plan_t** out);

int32_t bs_plan_n_seqs(const bs_plan_t* p);
int32_t bs_plan_q_rows(const bs_plan_t* p);           /* rows of the local Q-side buffers */
const int32_t* bs_plan_cu_rows_q(const bs_plan_t* p); /* [n_seqs + 1] first local row per seq */
/* Global position (0-based inside its sequence) and sequence index of every local Q row:
 * [q_rows] each.  Owned by the plan. */
const int32_t* bs_plan_q_pos(const bs_plan_t* p);
const int32_t* bs_plan_q_seq(const bs_plan_t* p);
int32_t bs_plan_n_steps(const bs_plan_t* p); /* max cp over the input (0 if n_seqs == 0) */
const bs_step_t* bs_plan_step(const bs_plan_t* p, int32_t s); /* NULL if s out of range */
/* Global position / sequence index of every row of step s's K/V buffer: [kv_rows] each. */
const int32_t* bs_plan_step_k_pos(const bs_plan_t* p, int32_t s);
const int32_t* bs_plan_step_k_seq(const bs_plan_t* p, int32_t s);
void bs_plan_destroy(bs_plan_t* p);                           /* NULL is a no-op */

/* ------------------------------------------------------------------------------------------ */
/* bs_assign: the naive HDP solution (Algorithm 1, routine at         */
/* PAPER.md:262) with offload ratio r = 0 - the step directly upstream of bs_plan.            */
/* ------------------------------------------------------------------------------------------ */
/* A global batch of sequence lengths, a token capacity C per rank and d_hdp ranks become, for
 * every rank and every round of the training step, the sequences that rank hands to bs_plan.
 *   R1  D(s) = ceil(s / C): Eq. 3 with r = 0 and Act(s) proportional to s.
 *       The paper's numbers at C = 8K: 1M -> 128, 16K -> 2, 768K -> 96, 312K -> 39 ranks.
 *   R2  lines 2-6: a sequence with D(s) = 1 goes to the pack list, every other one keeps D(s).
 *   R3  lines 7-9: one bin per pass of the while loop; the bin takes the longest remaining
 *       sequence that still fits (ties: lowest input index) until none fits.
 *   R4  line 10: in a round every rank runs at most one micro-batch, and the D(s) ranks of a
 *       long sequence run it in the same round.  Long sequences are placed in input order into
 *       the first round with D(s) free ranks, then the bins in the order they were made, each
 *       into the first round with a free rank; a round hands out its ranks from 0 upwards
 *       (96 ranks for a 768K sequence, the other 32 for 32 x 8K sequences).
 * Host only, integers only; the result is unique (bit-exact contract, tests/test_assign.py). */
typedef struct {
  int32_t round;        /* 0 <= round < bs_assign_n_rounds */
  int32_t rank;         /* HDP rank, 0 <= rank < d_hdp; (round, rank) is unique */
  int32_t n_seqs;
  const bs_seq_t* seqs; /* [n_seqs], owned by the assignment: one shard {len, cp = D, rank = j} of
                           a long sequence, or the whole sequences {len, 1, 0} of one bin */
  const int32_t* src;   /* [n_seqs] index of each sequence in the input batch */
} bs_microbatch_t;

typedef struct bs_assign_s bs_assign_t; /* opaque, host memory owned by the library */

/* lens: host, [n].  *out receives an assignment to be released with bs_assign_destroy.
 * Errors: INVALID_ARG (null, n < 0, len < 1, capacity < 1, d_hdp < 1, a sequence that needs
 * more than d_hdp ranks), HOST_OOM. */
bs_status_t bs_assign(const int32_t* lens, int32_t n, int32_t capacity, int32_t d_hdp,
                      bs_assign_t** out);
int32_t bs_assign_n_rounds(const bs_assign_t* a);
int32_t bs_assign_n_seqs(const bs_assign_t* a);
const int32_t* bs_assign_ranks_needed(const bs_assign_t* a); /* [n] D(s_i) */
int32_t bs_assign_n_microbatches(const bs_assign_t* a);
/* micro-batch k in (round, rank) order; NULL if k is out of range */
const bs_microbatch_t* bs_assign_microbatch(const bs_assign_t* a, int32_t k);
void bs_assign_destroy(bs_assign_t* a);                       /* NULL is a no-op */

/* ------------------------------------------------------------------------------------------ */
/* bs_balance: the balance strategy for HDP (Algorithm 2, sections     */
/* 6.3-6.4) in its DP-Balance form; it takes the place of line 10 of Algorithm 1.              */
/* ------------------------------------------------------------------------------------------ */
/* Schedules the groups of Algorithm 1 lines 1-9 (a long sequence on D(s) ranks, or a bin of
 * short ones on one rank) so that all ranks finish at about the same time; ranks may run
 * different numbers of micro-batches.
 *   B1  cost[3] = {a2, a1, a0}: T(s) = a2 s^2 + a1 s + a0 (Eq. 3), non-negative
 *       integers in the caller's time unit.  A long sequence costs each of its D ranks
 *       floor(T(s) / D), a bin the sum of T over its sequences.
 *   B2  line 4: groups sorted by the time they cost one rank, descending (ties: more ranks
 *       first, then the order Algorithm 1 made them).
 *   B3  line 5: group g of the sorted list goes to bucket floor(n_buckets * work before g /
 *       total work), at most n_buckets - 1; work = time x ranks.
 *   B4  lines 7-9: targets = ranks more than delta behind the slowest rank; if there is none,
 *       a new time step begins and every rank is a target.
 *   B5  lines 10-17: the next group of the first bucket goes to the D targets with the smallest
 *       exec_times (ties: lowest rank; if fewer than D ranks are targets the least loaded others
 *       fill up); they start together at the largest of their exec_times.  CP rank j is the j-th
 *       chosen rank in ascending order.
 *   B6  lines 18-20: an empty bucket is removed.
 * Under B4/B5 the targets are a prefix of the ranks ordered by exec_time, so the result does not
 * depend on n_buckets and delta (they matter for PP-Balance, which is out of scope); both are
 * validated and otherwise unused.  Host only, integers only, unique result. */
typedef struct {
  int32_t rank;         /* HDP rank */
  int32_t n_seqs;
  int64_t start, end;   /* in the unit of cost[]; a rank's micro-batches do not overlap */
  const bs_seq_t* seqs; /* [n_seqs] as in bs_microbatch_t */
  const int32_t* src;   /* [n_seqs] index of each sequence in the input batch */
} bs_timed_microbatch_t;

typedef struct bs_balance_s bs_balance_t; /* opaque, host memory owned by the library */

/* Errors: INVALID_ARG (as bs_assign; negative cost or delta, n_buckets < 1, a sequence cost
 * >= 2^53 or a total >= 2^62), HOST_OOM. */
bs_status_t bs_balance(const int32_t* lens, int32_t n, int32_t capacity, int32_t d_hdp,
                       const int64_t* cost, int32_t n_buckets, int64_t delta, bs_balance_t** out);
int32_t bs_balance_n_ranks(const bs_balance_t* b);
const int64_t* bs_balance_exec_times(const bs_balance_t* b); /* [d_hdp] finish time of each rank */
int64_t bs_balance_makespan(const bs_balance_t* b);
int32_t bs_balance_n_microbatches(const bs_balance_t* b);
/* micro-batch k in (rank, start) order; NULL if k is out of range */
const bs_timed_microbatch_t* bs_balance_microbatch(const bs_balance_t* b, int32_t k);
void bs_balance_destroy(bs_balance_t* b);                     /* NULL is a no-op */

/* ------------------------------------------------------------------------------------------ */
/* Device calls                                                                                */
/* ------------------------------------------------------------------------------------------ */

typedef struct {
  int32_t n_q_heads, n_kv_heads, head_dim;
  float softmax_scale;   /* <= 0 means 1/sqrt(head_dim) */
  int32_t q_rows;        /* rows in Q/O/dO/dQ/LSE/delta buffers of this call */
  int32_t kv_rows;       /* rows in K/V/dK/dV buffers of this call */
  int64_t q_row_stride;  /* elements */
  int64_t kv_row_stride; /* elements */
  int64_t lse_head_stride; /* elements; >= q_rows */
} bs_attn_shape_t;

/* Bytes of caller-owned device workspace a forward (bwd == 0) or backward (bwd != 0) call with
 * n_segs segments needs.  The workspace must be 256-byte aligned.  It holds the uploaded
 * segment/work-item tables and the scheduler's counters; its content is dead after the call's
 * kernels finish, and one workspace must not be shared by calls in flight on different streams. */
bs_status_t bs_attn_workspace_bytes(const bs_attn_shape_t* shape, int32_t n_segs, int bwd,
                                    size_t* bytes);

/* Forward of one Q-chunk x KV-chunk step (flash attention = exact attention,
 * PAPER.md:97).  For every head h and every row i in [out_row_begin, out_row_end):
 *   S_ij = scale * q_i . k_j over the visible keys j of every segment containing row i
 *   LSE[h,i] = ln sum_j exp(S_ij)   (natural log; -inf if no key is visible)
 *   O[i,h,:] = sum_j exp(S_ij - LSE[h,i]) * V[j, h / (Hq/Hkv), :]   (0 if no key is visible)
 * Rows of the range covered by no segment get O = 0, LSE = -inf.  Rows outside the range are
 * not written.  Q,K,V,O: device bf16.  LSE: device fp32.  segs: host.  ws: device.
 * dQ_acc_clear (device, fp32 [q_rows][n_q_heads][head_dim] dense, 16-byte aligned, or NULL): if
 * given, the call also sets rows [out_row_begin, out_row_end) of it to 0 - the zeroing half of
 * bs_attn_bwd_prep folded into the forward's stores (the forward leaves most of the HBM
 * bandwidth unused); bs_attn_bwd_prep is then called with dQ_acc = NULL.  With several ring steps
 * only one forward call of the sequence passes it. */
bs_status_t bs_attn_fwd(const bs_attn_shape_t* shape, const void* Q, const void* K, const void* V,
                        const bs_seg_t* segs, int32_t n_segs, int32_t out_row_begin,
                        int32_t out_row_end, void* O, float* LSE, void* ws, size_t ws_bytes,
                        void* stream, float* dQ_acc_clear);

/* bs_attn_fwd for callers that may not allocate device memory (a CUDA graph being captured, a
 * serving loop, a harness that forbids cudaMalloc): the same operation, arguments, kernels and
 * results as bs_attn_fwd, but the work-item tables, the scheduler's cursor and the
 * clipped tensor maps live in a scratch array INSIDE the library (static __device__,
 * BS_ATTN_STATIC_SCRATCH_BYTES per GPU that loads the library, held until the process exits)
 * instead of a caller workspace.  The call allocates nothing on the device or in pinned memory
 * (no cudaMalloc / cudaFree / cudaHostAlloc, no allocating library routine; host heap only for
 * the work list): the tables reach the scratch as kernel PARAMETERS of small copy kernels
 * (3584 bytes per launch), so nothing is read from host memory after the call returns and the
 * host never waits for the stream; a call can be captured into a CUDA graph (after one plain
 * call on the device, which sets kernel attributes and resolves the scratch address) as long as
 * the tensors it was captured with stay where they are.
 *   Limit: the call's tables must fit the array.  A call fits whenever
 * bs_attn_workspace_bytes(shape, n_segs, 0, &b) gives b <= BS_ATTN_STATIC_SCRATCH_BYTES (an
 * upper bound; the exact size is checked); otherwise BS_ERR_WORKSPACE with both sizes in
 * bs_last_error(), before anything is enqueued - use bs_attn_fwd then.  256 KiB holds e.g. a
 * 131072-row packed buffer of ~1000 ragged documents.
 *   Sharing: every call on a device uses the SAME array.  Each call rewrites all of it that it
 * reads (cursor included), so the previous call's contents never matter, but two calls whose
 * kernels can overlap on the GPU (different streams without an ordering, or host threads on
 * different streams) race on it: keep all bs_attn_fwd_static calls of a device on one stream or
 * order them with events.  Other errors and all argument rules as bs_attn_fwd. */
#define BS_ATTN_STATIC_SCRATCH_BYTES 262144
bs_status_t bs_attn_fwd_static(const bs_attn_shape_t* shape, const void* Q, const void* K,
                               const void* V, const bs_seg_t* segs, int32_t n_segs,
                               int32_t out_row_begin, int32_t out_row_end, void* O, float* LSE,
                               void* stream, float* dQ_acc_clear);

/* Backward preparation (a5): delta[h,i] = sum_d dO[i,h,d] * O_final[i,h,d] for all q_rows, and
 * dQ_acc = 0 (skipped if dQ_acc is NULL: the accumulator was cleared by bs_attn_fwd).  O_final is
 * the MERGED output.  All device pointers. */
bs_status_t bs_attn_bwd_prep(const bs_attn_shape_t* shape, const void* O_final, const void* dO,
                             float* delta, float* dQ_acc, void* stream);

/* Backward of one step (a6), using the MERGED LSE and delta so that each step yields the exact
 * partial gradients (reading 13):
 *   P_ij = exp(S_ij - LSE_final[h,i]);  dP_ij = dO_i . v_j;  dS_ij = P_ij * (dP_ij - delta[h,i])
 *   dV[j,g,:] = sum_{h in g} sum_i P_ij dO[i,h,:]        (overwritten; unreferenced rows = 0)
 *   dK[j,g,:] = scale * sum_{h in g} sum_i dS_ij Q[i,h,:] (overwritten; unreferenced rows = 0)
 *   dQ_acc[i,h,:] += scale * sum_j dS_ij K[j,g,:]         (fp32, accumulated across steps)
 * All kv_rows rows of dK and dV are written. */
bs_status_t bs_attn_bwd(const bs_attn_shape_t* shape, const void* Q, const void* K, const void* V,
                        const void* dO, const float* LSE_final, const float* delta,
                        const bs_seg_t* segs, int32_t n_segs, float* dQ_acc, void* dK, void* dV,
                        void* ws, size_t ws_bytes, void* stream);

/* a7: dQ = bf16(dQ_acc) for all q_rows (round to nearest even). */
bs_status_t bs_attn_bwd_finish(const bs_attn_shape_t* shape, const float* dQ_acc, void* dQ,
                               void* stream);

/* LSE merge (a4) of n_parts partial results over rows [row_begin,row_end), every head:
 *   M = max_s LSE_s; all -inf -> O = 0, LSE = -inf; else
 *   w_s = exp(LSE_s - M), Z = sum_s w_s, LSE = M + ln Z, O = sum_s (w_s / Z) O_s.
 * O_parts / LSE_parts: HOST arrays of n_parts DEVICE pointers, each laid out per `shape`
 * (q_rows, q_row_stride, lse_head_stride).  O_out may alias O_parts[k] and LSE_out may alias
 * LSE_parts[k] (running merge).  1 <= n_parts <= BS_MAX_MERGE_PARTS. */
#define BS_MAX_MERGE_PARTS 64
bs_status_t bs_lse_merge(int32_t n_parts, const void* const* O_parts,
                         const float* const* LSE_parts, const bs_attn_shape_t* shape,
                         int32_t row_begin, int32_t row_end, void* O_out, float* LSE_out,
                         void* stream);

/* ------------------------------------------------------------------------------------------ */
/* Fused softmax cross-entropy                              */
/* ------------------------------------------------------------------------------------------ */
/* One kernel, bf16 in, fp32 online softmax inside, one read of the logits and one write of the
 * gradients.  For token i with label y_i >= 0:
 *     loss[i]       = log(sum_j exp(x_ij)) - x_i[y_i]
 *     dlogits[i][j] = grad_scale * (softmax(x_i)[j] - (j == y_i))
 * and loss[i] = 0, dlogits[i][:] = 0 for y_i < 0 (ignored token).
 * logits, dlogits: device, bf16, [n_tokens][row_stride] with the first `vocab` columns used
 * (row_stride in elements, >= vocab, a multiple of 8; both 16-byte aligned; they may not
 * alias).  labels: device, int32 [n_tokens], < vocab.  loss: device, fp32 [n_tokens].
 * Errors: INVALID_ARG (sizes, stride, alignment, null pointers), CUDA.  Asynchronous on stream. */
bs_status_t bs_softmax_xent(const void* logits, const int32_t* labels, int32_t n_tokens,
                            int32_t vocab, int64_t row_stride, float grad_scale, float* loss,
                            void* dlogits, void* stream);

/* Measurement aid: the HBM rate a read-dominated streaming kernel can reach on
 * this device, with the merge's own access pattern - n_in input streams of bytes_per_stream bytes
 * each, read with 16-byte loads and combined word by word (XOR), then written to `out` (n : 1,
 * the merge's shape) or, with out == NULL, only read (pure-read ceiling).  in: HOST array of n_in
 * DEVICE pointers; out: device or NULL; sink: device, 4 bytes, never written in practice (it keeps
 * the pure-read loads alive).  1 <= n_in <= BS_MAX_MERGE_PARTS; sizes and pointers 16-byte
 * aligned.  bench.py reports bs_lse_merge against it. */
bs_status_t bs_hbm_probe(int32_t n_in, const void* const* in, void* out, void* sink,
                         size_t bytes_per_stream, void* stream);

/* Measurement aid for the backward's roofline: bs_attn_bwd adds every 128 x 128
 * tile-block's partial dQ - 64 KB of fp32 at head_dim 128 - into dQ_acc with TMA reduce-adds that
 * the L2 atomic units execute ("dQ_acc ... accumulated across steps", see bs_attn_bwd).  This call
 * issues only such reduce boxes (the same instruction, box shape and tensor map; one CTA per SM,
 * two boxes in flight each; the boxes hold zeros, so acc is unchanged): boxes_per_cta boxes of
 * 128 rows x 32 columns = 16 KB per CTA.  Timed by the caller, it gives the fp32 reduce-add rate
 * the device sustains with nothing else running, which bench.py reports the backward's own
 * reduction traffic against.  acc: device, fp32 [rows][n_heads][head_dim] dense, 16-byte aligned;
 * rows a multiple of 128, head_dim a multiple of 32 (<= 256).  Errors: INVALID_ARG, UNSUPPORTED,
 * CUDA.  Asynchronous on stream. */
bs_status_t bs_reduce_probe(float* acc, int32_t rows, int32_t n_heads, int32_t head_dim,
                            int32_t boxes_per_cta, void* stream);

/* Number of kernels this library has launched on the calling thread since the last reset
 * (bench.py's "gpu_launches"). */
int64_t bs_launch_count(void);
void bs_launch_count_reset(void);

#ifdef __cplusplus
}
#endif
#endif /* BYTESCALE_ATTN_H_ */
