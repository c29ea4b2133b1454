/* fcp.h — C ABI of libfcp: the per-CP-rank hot path of FlashCP (arxiv/paper_2606_08476),
 * B200 / sm_100a.  plan -> rank layout -> sharding-aware KV gather -> document-masked causal
 * attention forward/backward -> partial-result (LSE) merge; plus the dK/dV scatter-add (the
 * ReduceScatter stand-in, section 2) and the local / prefix split of a rank's keys (section 2b).
 *
 * Conventions (section 3.1): documents D=[d_0..d_{n-1}] packed in this order into a
 * context of C = sum d_k tokens; CP size N ("ranks"); a shard = (doc, start p, len s, rank) =
 * tokens [p, p+s) of one document; W(p,s) = (2p+s+1)*s/2.
 *
 * General rules
 *  - Every function returns an int: FCP_OK (0) or a negative fcp_status.  Nothing throws or
 *    aborts across this boundary (host allocation failures come back as FCP_NO_MEMORY).  The
 *    library keeps no mutable state of its own besides the objects it hands out: the only
 *    process-wide data are write-once caches of immutable facts (the SM count per device, the
 *    address of the driver's tensor-map encoder), published with atomics, so every entry point
 *    may be called from several threads and for several devices.  Objects are not internally
 *    synchronised: do not destroy one while another thread uses it.  One exception, stated at
 *    its declaration: fcp_attn_bwd_static works on a static device array shared by all of its
 *    calls on a device.
 *  - "host" pointers are ordinary CPU memory; "device" pointers are CUDA device memory of the
 *    current device.  The library owns only the opaque host objects it creates (fcp_plan,
 *    fcp_sched).  It never allocates, frees or synchronises device memory: inputs, outputs
 *    and workspace are the caller's (fcp_attn_bwd_static: the workspace is that static array), every device call is asynchronous on `stream`
 *    (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *  - Device tensors are bf16, row-major contiguous, "token-major varlen":
 *        q, o, dO, dq : [n_q , Hq , D]        k, v, dk, dv : [n_kv, Hkv, D]
 *        lse          : [Hq, n_q] float32 = natural log of sum_j exp(scale * q.k_j)
 *    D in {64, 128}; Hq % Hkv == 0; all base pointers 16-byte aligned.
 */
#ifndef FCP_H_
#define FCP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  FCP_OK = 0,
  FCP_INVALID_ARG = -1,      /* null pointer, n_ranks<1, n_docs<1, d_k<1, C % N != 0, R<1, bad index */
  FCP_UNSUPPORTED = -2,      /* D not in {64,128}, Hq % Hkv != 0, unknown dtype/strategy */
  FCP_BUFFER_TOO_SMALL = -3, /* required element count is written to *n_out */
  FCP_CUDA = -4,             /* a CUDA runtime/driver call or kernel launch failed */
  FCP_MISALIGNED = -5,       /* a device pointer or row pitch is not 16-byte aligned */
  FCP_NO_MEMORY = -6,        /* a host allocation failed (std::bad_alloc is caught at the boundary) */
  FCP_TOO_LARGE = -7         /* fcp_attn_bwd_static: the schedule's workspace exceeds
                                FCP_STATIC_WORKSPACE_BYTES */
} fcp_status;

const char* fcp_strerror(int status);

/* ------------------------------------------------------------------------------------------
 * 1. Sharding plan — Algorithm 1, host, integer arithmetic only.
 * ------------------------------------------------------------------------------------------ */
typedef struct fcp_plan fcp_plan;               /* opaque, host memory, owned by the library */

typedef struct { int32_t doc, start, len, rank; } fcp_shard;

enum { FCP_STRATEGY_HYBRID = 0,                 /* Algorithm 1: Whole-Doc + Per-Doc */
       FCP_STRATEGY_ALL_PER_DOC = 1,            /* every document in 2N chunks */
       FCP_STRATEGY_WHOLE_DOC = 2,              /* Whole-Doc sharding only */
       FCP_STRATEGY_PER_SEQ = 3 };              /* baseline: Llama3 CP, the packed sequence in 2N
                                                   chunks regardless of documents;
                                                   needs C % 2N == 0 */

typedef struct {
  int64_t imbalance_ppm;   /* target R = max/avg workload times 1e6; >= 1000000;
                              0 selects the default 1050000 */
  int32_t strategy;        /* FCP_STRATEGY_* */
  int32_t align_tokens;    /* 0 or 1: Algorithm 1 as read in DESIGN.md section 2.3.  A > 1: the
                              tile-aligned variant (ragged
                              shards cost kernel efficiency): Per-Doc chunk lengths are multiples
                              of A and chunks start on multiples of A (the < A leftover tokens
                              are a movable item at the document's end, next to the last chunk);
                              the equal-token repair cuts multiples of A from items that start
                              on a multiple of A and takes the < A remainder Eq. 2 forces from
                              the head of the donor's shortest item.  Ignored by
                              FCP_STRATEGY_PER_SEQ.  A = 128 matches the attention tiles. */
} fcp_plan_opts;

/* Builds the plan for documents `doc_lengths[0..n_docs)` (host) on `n_ranks` workers.
 * Deterministic: fixed tie-breaks.  opts == NULL selects the defaults.
 * Requires sum(doc_lengths) % n_ranks == 0 (Eq. 2).  *out must be released with
 * fcp_plan_destroy. */
int  fcp_plan_create(const int32_t* doc_lengths, int32_t n_docs, int32_t n_ranks,
                     const fcp_plan_opts* opts, fcp_plan** out);
void fcp_plan_destroy(fcp_plan* plan);

/* Canonical shard list, sorted by (rank, doc, start), contiguous neighbours merged.
 * rank == -1 selects all ranks.  Writes min(count, cap) entries to `out` (host, may be NULL when
 * cap == 0) and the full count to *n_out; returns FCP_BUFFER_TOO_SMALL when count > cap. */
int  fcp_plan_shards(const fcp_plan* plan, int32_t rank, fcp_shard* out, int32_t cap,
                     int32_t* n_out);
/* Ids of the documents Algorithm 1 moved to Per-Doc sharding, in the order they were popped
 * (descending length).  Same buffer protocol as fcp_plan_shards. */
int  fcp_plan_perdoc(const fcp_plan* plan, int32_t* doc_ids, int32_t cap, int32_t* n_out);

typedef struct {
  int32_t  n_ranks, n_docs, n_shards, n_per_doc, n_passes, reserved;
  int64_t  context_len;          /* C */
  int64_t  tokens_per_rank;      /* C / N (Eq. 2) */
  uint64_t max_load, sum_load;   /* max_j and sum_j of sum_i x_ij W_i (Eq. 3) */
  int64_t  imbalance_ppm;        /* floor(1e6 * max_load * N / sum_load) */
  int64_t  eq4_tokens;           /* (C/N)(N-1): static full-KV exchange (Eq. 4) */
  int64_t  eq5_tokens;           /* (N-1) max_j sum_{i in S-hat} x_ij s_i (Eq. 5) */
  int64_t  max_remote_tokens, sum_remote_tokens;     /* exact KV rows a rank needs from others */
  int64_t  max_gathered_tokens, sum_gathered_tokens; /* rows of the rank's gathered KV buffer */
} fcp_stats;
int  fcp_plan_stats(const fcp_plan* plan, fcp_stats* out);

typedef struct {
  int32_t  n_shards, n_segs;     /* shards on the rank; documents (KV segments) it has queries of */
  int64_t  n_q;                  /* local query rows = C/N */
  int64_t  n_kv;                 /* gathered KV rows = sum_k E_r(k) */
  int64_t  remote_tokens;        /* gathered rows owned by another rank */
  int64_t  nonlast_tokens;       /* sum of s_i over the rank's shards in S-hat */
  uint64_t load;                 /* sum of W_i on the rank */
} fcp_rank_stats;
int  fcp_plan_rank_stats(const fcp_plan* plan, int32_t rank, fcp_rank_stats* out);

/* Varlen descriptors of one rank.  All arrays are caller-allocated HOST int32 arrays sized from
 * fcp_plan_rank_stats (a NULL array is skipped).  Local query rows are the rank's shards in
 * (doc, start) order; KV segment g holds tokens [0, E_r(k)) of the g-th document (ascending k)
 * with a query on the rank, E_r(k) = max(p+s) over the rank's shards of k. */
typedef struct {
  int32_t* cu_seqlens_q;    /* [n_shards+1] local row offsets of the shards */
  int32_t* q_pos_off;       /* [n_shards]   p_i: document position of the shard's first query */
  int32_t* shard_seg;       /* [n_shards]   KV segment the shard reads */
  int32_t* cu_seqlens_k;    /* [n_segs+1]   row offsets of the segments in the gathered buffer */
  int32_t* kv_src_start;    /* [n_segs]     global token offset off_k of the segment's document */
  int32_t* kv_len;          /* [n_segs]     E_r(k) */
  int32_t* q_token_index;   /* [n_q]        global token of every local query row */
  int32_t* kv_token_index;  /* [n_kv]       global token of every gathered KV row */
} fcp_layout;
int  fcp_rank_layout(const fcp_plan* plan, int32_t rank, fcp_layout* out);

/* ------------------------------------------------------------------------------------------
 * 2. Sharding-aware KV gather (the "data copy" of PAPER.md:255).
 *    Copies, for every document k with a query on `rank`, rows [off_k, off_k + E_r(k)) of the
 *    global K and V [C, Hkv, D] (device) into the contiguous k_out, v_out [n_kv, Hkv, D]
 *    (device).  One kernel launch.  On one GPU this stands in for "receive + copy": the bytes
 *    a real CP group would communicate are counted in *counts (host, may be NULL), never sent.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
  int64_t total_tokens, remote_tokens;   /* rows copied; rows owned by another rank */
  int64_t total_bytes, remote_bytes;     /* K and V together, one pass */
  int32_t n_ranges, reserved;            /* contiguous source ranges after merging neighbours */
} fcp_gather_counts;
int  fcp_kv_gather(const fcp_plan* plan, int32_t rank, const void* K, const void* V,
                   void* k_out, void* v_out, int32_t n_kv_heads, int32_t head_dim,
                   void* stream, fcp_gather_counts* counts);

/* dKV reduction of one rank (the gradients of the communicated KV go back to
 * the ranks that own the tokens; the inverse of the KV selection of PAPER.md:111-113; SURVEY.md
 * section 8(f) NEXT 1).  Adds the rank's own contribution dk_r, dv_r [n_kv, Hkv, D] (device,
 * layout of the gathered k, v as written by fcp_attn_bwd; src_dtype FCP_DTYPE_BF16 or
 * FCP_DTYPE_F32) into the global fp32 accumulators dK, dV [C, Hkv, D] (device): row i of the
 * rank's buffer is added to global token kv_token_index[i].  The rows of one rank are distinct
 * tokens, so one call needs no atomics; calls for different ranks must be ordered on the stream
 * (virtual ranks) — across real GPUs this is the ReduceScatter the bytes of which *counts
 * reports.  One kernel launch, asynchronous on `stream`. */
int  fcp_kv_scatter_add(const fcp_plan* plan, int32_t rank, const void* dk_r, const void* dv_r,
                        int32_t src_dtype, float* dK, float* dV, int32_t n_kv_heads,
                        int32_t head_dim, void* stream, fcp_gather_counts* counts);

/* Last step of the dKV reduction: the fp32 accumulators dK, dV (device, n_elems = C*Hkv*D each,
 * filled by fcp_kv_scatter_add over all ranks) rounded to nearest-even bf16 into dK_out, dV_out
 * (device, same shape): the tensors the owner of the tokens hands on.  n_elems
 * must be a multiple of 8 and all pointers 16-byte aligned.  One kernel launch, asynchronous. */
int  fcp_kv_reduce_finish(const float* dK, const float* dV, void* dK_out, void* dV_out,
                          int64_t n_elems, void* stream);

/* ------------------------------------------------------------------------------------------
 * 2b. Local / prefix split of a rank's keys.  PAPER.md:15 and
 *    PAPER.md:234 describe the communication-hiding alternative: compute on the keys a worker
 *    already holds while the others travel, then aggregate the partial results.
 *    Per shard (k, p, s) of the rank:
 *      FCP_PIECE_LOCAL  : the shard's own tokens [p, p+s), causal inside the shard — needs no
 *                         byte from another rank (its buffer is the rank's own K/V rows in
 *                         local query order);
 *      FCP_PIECE_PREFIX : the tokens [0, p) before it, all visible to every row.
 *    The two key sets are disjoint and their union is the prefix [0, p+s) the unsplit path
 *    (FCP_PIECE_FULL) attends to, so  fcp_merge(fwd(LOCAL), fwd(PREFIX))  equals the unsplit
 *    forward; the backward of each piece takes the merged o / lse, dq accumulates over the
 *    pieces (fcp_attn_args.dq_accum) and dK / dV scatter-add per piece.
 *    In both pieces every shard is its own KV segment (n_segs = n_shards, zero-length segments
 *    allowed); a prefix two shards of the rank share appears once per shard in the PREFIX
 *    buffer, and fcp_rank_stats.remote_tokens / counts->remote_* still count each distinct
 *    remote token once (LOCAL: 0, PREFIX: the unsplit gather's).  The *_piece entry points with
 *    FCP_PIECE_FULL are the plain ones.
 * ------------------------------------------------------------------------------------------ */
enum { FCP_PIECE_FULL = 0, FCP_PIECE_LOCAL = 1, FCP_PIECE_PREFIX = 2 };
int  fcp_plan_piece_stats(const fcp_plan* plan, int32_t rank, int32_t piece, fcp_rank_stats* out);
int  fcp_piece_layout(const fcp_plan* plan, int32_t rank, int32_t piece, fcp_layout* out);
int  fcp_kv_gather_piece(const fcp_plan* plan, int32_t rank, int32_t piece, const void* K,
                         const void* V, void* k_out, void* v_out, int32_t n_kv_heads,
                         int32_t head_dim, void* stream, fcp_gather_counts* counts);
/* Rows of a PREFIX buffer can name the same global token twice (two shards of one document on
 * the rank); such ranges are added by separate, stream-ordered launches — still no atomics. */
int  fcp_kv_scatter_add_piece(const fcp_plan* plan, int32_t rank, int32_t piece, const void* dk_r,
                              const void* dv_r, int32_t src_dtype, float* dK, float* dV,
                              int32_t n_kv_heads, int32_t head_dim, void* stream,
                              fcp_gather_counts* counts);

/* ------------------------------------------------------------------------------------------
 * 3. Tile schedule of one rank: the (shard, q-tile, head) / (segment, kv-tile, kv-head) work
 *    lists of the attention kernels, ordered by descending cost so that short shards do not
 *    starve the SMs.  Host object; fcp_sched_upload copies the lists into
 *    caller-provided device workspace once per (plan, rank).
 *    Row t of shard i sees keys j of its segment with  j <= q_pos_off[i] + t  and
 *    j < cu_seqlens_k[g+1]-cu_seqlens_k[g]  (q_pos_off may be negative when the segment is a
 *    KV *piece* that starts after the document's first token; rows that see no key produce
 *    o = 0, lse = -inf).
 * ------------------------------------------------------------------------------------------ */
typedef struct fcp_sched fcp_sched;             /* opaque, host memory, owned by the library */
int  fcp_sched_create(const int32_t* cu_seqlens_q, const int32_t* q_pos_off,
                      const int32_t* shard_seg, int32_t n_shards,
                      const int32_t* cu_seqlens_k, int32_t n_segs,
                      int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                      fcp_sched** out);          /* all arrays host */
int  fcp_sched_from_plan(const fcp_plan* plan, int32_t rank, int32_t n_q_heads,
                         int32_t n_kv_heads, int32_t head_dim, fcp_sched** out);
int  fcp_sched_from_plan_piece(const fcp_plan* plan, int32_t rank, int32_t piece,
                               int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                               fcp_sched** out);             /* section 2b */
void fcp_sched_destroy(fcp_sched* sched);
/* Device bytes needed by fcp_sched_upload + fcp_attn_fwd + fcp_attn_bwd (work lists, tile
 * counters, backward scratch: padded (lse, delta) and the fp32 dq accumulator). */
int  fcp_sched_workspace_size(const fcp_sched* sched, size_t* device_bytes);
int  fcp_sched_upload(const fcp_sched* sched, void* workspace, void* stream);

typedef struct {
  int32_t n_fwd_items, n_bwd_items;   /* work items of the forward / backward kernels */
  int64_t fwd_kv_tiles;               /* (q-tile, kv-tile) pairs the forward computes, x heads */
  int64_t bwd_tile_pairs;             /* (kv-tile, q-tile) pairs the backward computes, x heads */
  uint64_t useful_pairs;              /* sum of unmasked (q,k) pairs over the rank's shards */
  int64_t n_q, n_kv;
  int64_t n_q_pad;                    /* query rows with every shard padded to a multiple of the
                                         backward's q tile: rows of fcp_attn_args.dq_accum */
} fcp_sched_info;
int  fcp_sched_get_info(const fcp_sched* sched, fcp_sched_info* out);

/* Read-back of the host work lists as int32 words (what fcp_sched_upload sends to the device;
 * for tests and tools).  `which`:
 *   FCP_LIST_FWD_ITEMS  8 words per item, grouped by CTA in processing order:
 *                       q_row0, q_rows, kv_row0, kv_len, q_pos0, n_kv_tiles, head0, kv_head
 *                       (one 128-row q tile of one shard x one pack of 1 or 2 query heads of one
 *                       kv head; KV tiles [0, n_kv_tiles) of 128 rows are visited, later tiles
 *                       are fully masked)
 *   FCP_LIST_BWD_ITEMS  8 words per item: kv_row0, kv_rows, kv_pos0, kv_head, sub_begin,
 *                       sub_end, n_iters, 0   (one 128-row KV tile of one segment x one kv head)
 *   FCP_LIST_BWD_SUBS   4 words per entry: q_row0, q_pos0, q_rows, pad_row0 (a shard seen by a
 *                       KV tile, from the first 64-row q tile that sees it to the shard's end)
 *   FCP_LIST_FWD_CTA / FCP_LIST_BWD_CTA   n_cta + 1 offsets: CTA c owns items [off[c], off[c+1])
 * Items are sorted by descending cost (n_kv_tiles + 1, n_iters + 2; stable in enumeration order:
 * shards, q tiles, kv heads, packs / segments, KV tiles, kv heads) and handed one by one to the
 * least loaded CTA, ties to the lowest CTA index.  Writes min(cap_words, n) words and the total
 * n to *n_words. */
enum { FCP_LIST_FWD_ITEMS = 0, FCP_LIST_BWD_ITEMS = 1, FCP_LIST_BWD_SUBS = 2, FCP_LIST_FWD_CTA = 3,
       FCP_LIST_BWD_CTA = 4 };
int  fcp_sched_get_list(const fcp_sched* sched, int32_t which, int32_t* out, int64_t cap_words,
                        int64_t* n_words);

/* ------------------------------------------------------------------------------------------
 * 4. Document-masked causal attention, forward and backward.
 *      forward : o = softmax(scale q K^T + mask) V, lse = log sum exp   (per shard, per head)
 *      backward: dV = P^T dO, dP = dO V^T, dS = P o (dP - rowsum(dO o O)),
 *                dQ = scale dS K, dK = scale dS^T Q; dk, dv summed over the G = Hq/Hkv query
 *                heads of a kv head; they hold only THIS rank's queries' contributions, in the
 *                layout of k, v (global dK = sum over ranks of scatter-add).
 *    bf16 tensor-core products with fp32 accumulation, fp32 softmax.
 *    Precondition: every row of q, k, v, dO handed to these calls holds finite values.  The
 *    kernels read 128-row boxes that run past the end of a segment or shard into its neighbour's
 *    rows and mask what they compute there: masked SCORES are replaced by selection, so the
 *    forward tolerates non-finite values in the K rows of a neighbouring segment
 *    (tests/test_gpu_parity.py::test_nonfinite_neighbour_keys), but a masked probability is an
 *    exact zero that still multiplies the neighbour's V row (forward) and K / V rows (backward)
 *    inside the tensor core, where 0 * Inf = NaN: a NaN or Inf in ANOTHER document's V, or in
 *    K / V during the backward, can reach the last 128-row tile of this one.
 * ------------------------------------------------------------------------------------------ */
enum { FCP_DTYPE_BF16 = 0, FCP_DTYPE_F32 = 1 };
typedef struct {
  const fcp_sched* sched;    /* host */
  void*       workspace;     /* device, >= fcp_sched_workspace_size bytes, uploaded */
  const void* q;             /* device bf16 [n_q , Hq , D] */
  const void* k;             /* device bf16 [n_kv, Hkv, D] */
  const void* v;             /* device bf16 [n_kv, Hkv, D] */
  void*       o;             /* device bf16 [n_q , Hq , D]: written by fwd, read by bwd */
  float*      lse;           /* device f32  [Hq, n_q]    : written by fwd, read by bwd */
  float       scale;         /* softmax scale, e.g. 1/sqrt(D) */
  int32_t     dkv_dtype;     /* element type of dk, dv written by fcp_attn_bwd: FCP_DTYPE_BF16 (0)
                                or FCP_DTYPE_F32 (partials that a dKV reduction sums in fp32) */
  void*       stream;
  void*       ev_start;      /* optional cudaEvent_t (NULL = none) recorded on `stream` right before */
  void*       ev_stop;       /* ... and right after the call's dominant kernel (the tcgen05
                                attention kernel of fwd / the main kernel of bwd): lets a caller
                                time that kernel alone without a profiler */
  float*      dq_accum;      /* fcp_attn_bwd only, optional (NULL = the workspace's own): device
                                f32 [Hq, n_q_pad, D] accumulator of UNSCALED dQ shared by the
                                backward calls over several KV pieces of the same queries
                                (section 2b; the pieces' schedules have the same n_q_pad) */
  int32_t     dq_flags;      /* FCP_DQ_* bits, only read when dq_accum != NULL */
} fcp_attn_args;
enum {
  FCP_DQ_KEEP = 1,           /* do not zero dq_accum first: it holds an earlier piece's partial */
  FCP_DQ_NO_OUTPUT = 2       /* do not convert to dq yet (dq may be NULL): more pieces follow */
};
int  fcp_attn_fwd(const fcp_attn_args* args);
int  fcp_attn_bwd(const fcp_attn_args* args, const void* dO, void* dq, void* dk, void* dv);

/* fcp_attn_bwd for callers that cannot provide a device workspace (code under CUDA graph capture,
 * serving loops and harnesses that forbid cudaMalloc): the same three kernels, with the work
 * lists, the (lse, delta) scratch and the fp32 dQ accumulator of the backward (the
 * formulas of this section) in a workspace the LIBRARY owns: a file-scope `static __device__`
 * array of FCP_STATIC_WORKSPACE_BYTES that every GPU which loads the library holds until the
 * process exits.  The call allocates and frees nothing on the host heap or the device.
 *   args->workspace must be NULL; every other field, dO, dq, dk, dv as for fcp_attn_bwd (inputs
 *   and outputs stay the caller's).  No fcp_sched_upload is needed: the call copies the
 *   schedule's lists into the static workspace on args->stream (from pageable host memory owned
 *   by the schedule), then launches fcp_bwd_prep, fcp_attn_bwd_main, fcp_bwd_dq_convert there.
 *   (That list copy is the one step a stream capture would refuse - capture takes no copy from
 *   pageable memory - and comes back as FCP_CUDA; the kernels themselves capture.)
 *   FCP_TOO_LARGE when fcp_sched_workspace_size(args->sched) > FCP_STATIC_WORKSPACE_BYTES
 *   (nothing is launched); roughly n_q_pad * Hq * (4 D + 8) bytes plus the lists, e.g. 2000 query
 *   rows at Hq = 32, D = 128 or 8000 at Hq = 8.
 *   The workspace keeps the previous call's contents; the call itself rewrites the lists and the
 *   scratch and zeroes the accumulator (fcp_bwd_prep), so nothing carries over.  All calls on a
 *   device share the one array: calls that overlap on the GPU (different streams, or several host
 *   threads launching on one device) RACE on it; order them on one stream or with events.  With a
 *   caller-owned args->dq_accum only the lists and the (lse, delta) scratch live there, the same
 *   rule applies. */
#define FCP_STATIC_WORKSPACE_BYTES (32u << 20)
int  fcp_attn_bwd_static(const fcp_attn_args* args, const void* dO, void* dq, void* dk, void* dv);

/* ------------------------------------------------------------------------------------------
 * 5. Partial-result aggregation: combines attention partials computed over
 *    two disjoint key sets:  lse = log(e^lse_a + e^lse_b),
 *    o = e^(lse_a-lse) o_a + e^(lse_b-lse) o_b.  A partial with lse = -inf has weight 0.
 *    o_* : [n_rows, n_heads, head_dim] (o_dtype: 0 = bf16, 1 = f32), lse_* : [n_heads, n_rows]
 *    f32.  Outputs may alias the `a` inputs.
 * ------------------------------------------------------------------------------------------ */
int  fcp_merge(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b,
               void* o_out, float* lse_out, int64_t n_rows, int32_t n_heads, int32_t head_dim,
               int32_t o_dtype, void* stream);

/* Library build information: "sm_100a;<git-less version string>". */
const char* fcp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FCP_H_ */
