// Internal (non-ABI) definitions shared by the host and device parts of libfcp.
#pragma once
#include <cstdint>
#include <new>
#include <vector>

#include "fcp.h"

struct fcp_plan {
  std::vector<int32_t> d;          // document lengths, packed order
  std::vector<int64_t> off;        // off[k] = sum_{k'<k} d[k'], off[n] = C
  int32_t n_ranks = 0;
  int64_t C = 0, T = 0;
  std::vector<fcp_shard> shards;   // canonical: (rank, doc, start), merged
  std::vector<int32_t> rank_begin; // [N+1] index range of each rank in `shards`
  std::vector<int32_t> per_doc;    // popped order
  int32_t n_passes = 0;
  uint64_t max_load = 0, sum_load = 0;
};

// One rank's view of the plan: local query order and KV prefix segments.
struct RankView {
  std::vector<int32_t> cu_q, q_pos_off, shard_seg, cu_k, kv_src_start, kv_len, seg_doc;
  int64_t n_q = 0, n_kv = 0, remote = 0, nonlast = 0;
  uint64_t load = 0;
};
// piece: FCP_PIECE_FULL (one segment per document prefix) or the local / prefix split (one
// segment per shard, fcp.h section 2b)
void fcp_build_rank_view(const fcp_plan& p, int32_t rank, RankView& v,
                         int32_t piece = FCP_PIECE_FULL);

inline uint64_t fcp_W(uint64_t p, uint64_t s) { return (2 * p + s + 1) * s / 2; }

// ---- tile schedule (host list + device pull) ------------------------------------------------
// Forward work item: one 128-row q tile of one shard for a pack of NQ query heads of one kv head.
struct FwdItem {
  int32_t q_row0;      // first local query row of the tile
  int32_t q_rows;      // valid rows (1..128)
  int32_t kv_row0;     // first row of the shard's KV segment in k/v
  int32_t kv_len;      // rows of the segment
  int32_t q_pos0;      // document position of the tile's first row (may be negative)
  int32_t n_kv_tiles;  // KV tiles [0, n_kv_tiles) of 128 rows to visit (0 = no visible key)
  int32_t head0;       // first query head of the pack
  int32_t kv_head;
};
// Backward work item: one 128-row KV tile of one segment for one kv head; loops over the
// (shard, q tile, query head) triples that see it.
struct BwdItem {
  int32_t kv_row0;     // first row of the KV tile in k/v (segment start + 128*tile)
  int32_t kv_rows;     // valid rows of the tile inside the segment (1..128)
  int32_t kv_pos0;     // document/segment position of the tile's first row
  int32_t kv_head;
  int32_t sub_begin;   // range into the BwdSub list
  int32_t sub_end;
  int32_t n_iters;     // total inner iterations = sum over subs of n_q_tiles * G
  int32_t reserved;
};
struct BwdSub {        // one shard seen by a KV tile
  int32_t q_row0;      // local row of the first q tile to visit
  int32_t q_pos0;      // document position of that row
  int32_t q_rows;      // valid rows from q_row0 to the shard's end
  int32_t pad_row0;    // row of the same tile in the padded (lse, delta) scratch
};

constexpr int FCP_TQ = 128;   // forward q-tile rows
constexpr int FCP_TK = 128;   // KV-tile rows (forward and backward)
constexpr int FCP_BQ = 64;    // backward q-tile rows

struct fcp_sched {
  int32_t Hq = 0, Hkv = 0, D = 0, G = 0, NQ = 1;   // NQ = query heads per forward CTA pack
  int64_t n_q = 0, n_kv = 0, n_q_pad = 0;          // n_q_pad: rows of the padded bwd scratch
  std::vector<int32_t> cu_q, q_pos_off, shard_seg, cu_k;
  std::vector<int32_t> shard_pad0;                 // [ns] first padded row of each shard
  std::vector<int32_t> tile_meta;                  // per padded 64-row tile: (local row0, valid rows)
  // Work lists, grouped by CTA: CTA c of the persistent grid walks fwd[fwd_cta_off[c] ..
  // fwd_cta_off[c+1]) in order (greedy longest-processing-time assignment, fcp_sched.cpp).
  int32_t n_cta = 0;
  std::vector<FwdItem> fwd;
  std::vector<BwdItem> bwd;
  std::vector<int32_t> fwd_cta_off, bwd_cta_off;   // [n_cta + 1]
  std::vector<uint8_t> image;                      // host image of workspace [0, off_lsed): one upload
  std::vector<BwdSub> bwd_sub;
  int64_t fwd_kv_tiles = 0, bwd_tile_pairs = 0;
  uint64_t useful_pairs = 0;
  // workspace layout (byte offsets, 256-byte aligned)
  size_t off_counters = 0, off_fwd = 0, off_bwd = 0, off_sub = 0, off_shard_meta = 0,
         off_fwd_cta = 0, off_bwd_cta = 0, off_lsed = 0, off_dq = 0, total = 0;
};

// Runs the body of an extern "C" entry point: nothing may throw across the C ABI (fcp.h), so a
// failed host allocation becomes FCP_NO_MEMORY and anything else FCP_INVALID_ARG.
template <class F>
int fcp_guard(F&& body) noexcept {
  try {
    return body();
  } catch (const std::bad_alloc&) {
    return FCP_NO_MEMORY;
  } catch (...) {
    return FCP_INVALID_ARG;
  }
}

// SM count of the current device (148 on B200; also the answer when no device is visible, e.g.
// a schedule built on a CPU-only box).  Write-once per-device cache behind atomics.
int32_t fcp_sm_count();
