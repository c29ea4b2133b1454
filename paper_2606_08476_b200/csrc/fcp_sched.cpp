// Tile schedule of one rank (host part): enumerates the forward (shard, q-tile, head-pack) and
// backward (segment, kv-tile, kv-head) work items, skips fully masked tiles and orders items by
// descending cost and assigns them to the persistent CTAs by greedy longest-processing-time, so
// that short shards do not starve the SMs (short shards lower kernel
// efficiency).  The assignment is static and deterministic; every CTA walks its own list.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstring>
#include <memory>
#include <new>

#include "fcp_internal.h"

namespace {
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Stable sort by descending integer key (counting sort: the keys are tile / iteration counts).
template <typename Item, typename Key>
void stable_sort_desc(std::vector<Item>& v, Key key) {
  int64_t mx = 0;
  for (const Item& x : v) mx = std::max<int64_t>(mx, key(x));
  std::vector<int32_t> pos((size_t)mx + 2, 0);
  for (const Item& x : v) ++pos[(size_t)(mx - key(x)) + 1];
  for (size_t i = 1; i < pos.size(); ++i) pos[i] += pos[i - 1];
  std::vector<Item> out(v.size());
  for (const Item& x : v) out[pos[(size_t)(mx - key(x))]++] = x;
  v.swap(out);
}

// Greedy longest-processing-time assignment of items (already sorted by descending cost) to
// n_cta persistent CTAs; `items` is permuted so that every CTA's list is contiguous (in the
// order the items were assigned) and cta_off[c] .. cta_off[c+1] delimits it.  Deterministic:
// the next item goes to the least loaded CTA, ties to the lowest CTA index.  Costs are small
// positive integers, so the priority queue is a bucket queue: bucket[l] = bit set of the CTAs
// with load l.  The least load never decreases (every cost is >= 1) and never exceeds
// avg + max cost, so one pointer walks the buckets once; taking the next CTA is a
// count-trailing-zeros.  (A binary heap of (load, cta) pairs gives the same lists at ~90 ns
// per item: 2/3 of the build time of a schedule of short documents.)  The permutation is a
// counting scatter.
template <typename Item, typename Cost>
void assign_lpt(std::vector<Item>& items, int32_t n_cta, Cost cost, std::vector<int32_t>& cta_off) {
  const size_t words = ((size_t)n_cta + 63) / 64;
  int64_t total = 0, mx = 1;
  for (const Item& x : items) {
    const int64_t c = cost(x);
    total += c;
    mx = std::max(mx, c);
  }
  const size_t n_buckets = (size_t)(total / n_cta + mx + 2);
  std::vector<uint64_t> bucket(n_buckets * words, 0);
  for (int32_t c = 0; c < n_cta; ++c) bucket[(size_t)c / 64] |= 1ull << (c % 64);   // all at load 0
  std::vector<int32_t> owner(items.size());
  cta_off.assign((size_t)n_cta + 1, 0);
  size_t lo = 0;                                  // least load with a CTA in its bucket
  for (size_t i = 0; i < items.size(); ++i) {
    size_t w = 0;
    for (;;) {
      for (w = 0; w < words && bucket[lo * words + w] == 0; ++w) {}
      if (w < words) break;
      ++lo;
    }
    uint64_t& word = bucket[lo * words + w];
    const int32_t c = (int32_t)(w * 64 + (size_t)__builtin_ctzll(word));
    word &= word - 1;
    owner[i] = c;
    ++cta_off[(size_t)c + 1];
    const size_t nl = lo + (size_t)cost(items[i]);
    bucket[nl * words + (size_t)c / 64] |= 1ull << (c % 64);
  }
  for (int32_t c = 0; c < n_cta; ++c) cta_off[(size_t)c + 1] += cta_off[c];
  std::vector<int32_t> pos(cta_off.begin(), cta_off.end() - 1);
  std::vector<Item> out(items.size());
  for (size_t i = 0; i < items.size(); ++i) out[(size_t)pos[owner[i]]++] = items[i];
  items.swap(out);
}
}

// Persistent grid size = SM count of the current device.  The attribute query costs more than
// the rest of a small schedule, so the answer is cached per device: a write-once table of
// immutable hardware facts behind atomics (safe from any thread, for any device).
int32_t fcp_sm_count() {
  constexpr int kMaxDev = 64;
  static std::atomic<int32_t> cache[kMaxDev];      // 0 = not queried yet
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return 148;                                    // no device visible (CPU-only box)
  }
  if (dev >= 0 && dev < kMaxDev) {
    const int32_t c = cache[dev].load(std::memory_order_relaxed);
    if (c > 0) return c;
  }
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) {
    cudaGetLastError();
    return 148;
  }
  if (dev >= 0 && dev < kMaxDev) cache[dev].store(n, std::memory_order_relaxed);
  return n;
}

// n_cta: size of the persistent grid
static int sched_create_impl(const int32_t* cu_seqlens_q, const int32_t* q_pos_off,
                        const int32_t* shard_seg, int32_t n_shards, const int32_t* cu_seqlens_k,
                        int32_t n_segs, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                        int32_t n_cta, fcp_sched** out) {
  if (!cu_seqlens_q || !q_pos_off || !shard_seg || !cu_seqlens_k || !out || n_shards < 0 ||
      n_segs < 0 || n_q_heads < 1 || n_kv_heads < 1)
    return FCP_INVALID_ARG;
  if ((head_dim != 64 && head_dim != 128) || n_q_heads % n_kv_heads != 0) return FCP_UNSUPPORTED;
  if (cu_seqlens_q[0] != 0 || cu_seqlens_k[0] != 0) return FCP_INVALID_ARG;
  for (int i = 0; i < n_shards; ++i)
    if (cu_seqlens_q[i + 1] < cu_seqlens_q[i] || shard_seg[i] < 0 || shard_seg[i] >= n_segs)
      return FCP_INVALID_ARG;
  for (int g = 0; g < n_segs; ++g)
    if (cu_seqlens_k[g + 1] < cu_seqlens_k[g]) return FCP_INVALID_ARG;

  std::unique_ptr<fcp_sched> owner(new fcp_sched());
  fcp_sched* s = owner.get();
  s->Hq = n_q_heads;  s->Hkv = n_kv_heads;  s->D = head_dim;
  s->G = n_q_heads / n_kv_heads;
  s->NQ = (s->G % 2 == 0) ? 2 : 1;
  s->cu_q.assign(cu_seqlens_q, cu_seqlens_q + n_shards + 1);
  s->q_pos_off.assign(q_pos_off, q_pos_off + n_shards);
  s->shard_seg.assign(shard_seg, shard_seg + n_shards);
  s->cu_k.assign(cu_seqlens_k, cu_seqlens_k + n_segs + 1);
  s->n_q = s->cu_q.back();
  s->n_kv = s->cu_k.back();

  // ---- forward items ----
  const int packs = s->G / s->NQ;
  s->shard_pad0.resize(n_shards);
  s->fwd.reserve((size_t)((s->n_q + FCP_TQ - 1) / FCP_TQ + n_shards) * s->Hkv * packs);
  int64_t pad = 0;
  for (int i = 0; i < n_shards; ++i) {
    const int32_t a = s->cu_q[i], len = s->cu_q[i + 1] - a, p = s->q_pos_off[i];
    const int32_t g = s->shard_seg[i];
    const int32_t kv0 = s->cu_k[g], kvl = s->cu_k[g + 1] - kv0;
    s->shard_pad0[i] = (int32_t)pad;
    pad += (int64_t)(len + FCP_BQ - 1) / FCP_BQ * FCP_BQ;
    // exact unmasked-pair count (statistic): sum over rows t of clamp(p + t + 1, 0, kvl) --
    // zero up to row t_lo, p + t + 1 up to row t_hi, kvl from there on
    if (kvl > 0 && len > 0) {
      const int64_t a = (int64_t)p + 1;
      const int64_t t_lo = std::min<int64_t>(len, std::max<int64_t>(0, 1 - a));
      const int64_t t_hi = std::min<int64_t>(len, std::max<int64_t>(t_lo, (int64_t)kvl - a));
      const int64_t m = t_hi - t_lo;
      s->useful_pairs += (uint64_t)(m * a + (t_lo + t_hi - 1) * m / 2 + (len - t_hi) * (int64_t)kvl);
    }
    for (int32_t r0 = 0; r0 < len; r0 += FCP_TQ) {
      FwdItem it;
      it.q_row0 = a + r0;
      it.q_rows = std::min(FCP_TQ, len - r0);
      it.kv_row0 = kv0;
      it.kv_len = kvl;
      it.q_pos0 = p + r0;
      const int64_t last_vis = std::min<int64_t>(kvl - 1, (int64_t)it.q_pos0 + it.q_rows - 1);
      it.n_kv_tiles = last_vis < 0 ? 0 : (int32_t)(last_vis / FCP_TK + 1);
      for (int hk = 0; hk < s->Hkv; ++hk)
        for (int pk = 0; pk < packs; ++pk) {
          it.kv_head = hk;
          it.head0 = hk * s->G + pk * s->NQ;
          s->fwd.push_back(it);
          s->fwd_kv_tiles += (int64_t)it.n_kv_tiles * s->NQ;
        }
    }
  }
  s->n_q_pad = pad;
  for (int i = 0; i < n_shards; ++i) {
    const int32_t a = s->cu_q[i], len = s->cu_q[i + 1] - a;
    for (int32_t r0 = 0; r0 < len; r0 += FCP_BQ) {
      s->tile_meta.push_back(a + r0);
      s->tile_meta.push_back(std::min(FCP_BQ, len - r0));
    }
  }
  stable_sort_desc(s->fwd, [](const FwdItem& x) { return (int64_t)x.n_kv_tiles; });
  s->n_cta = n_cta;
  // cost in KV-tile steps; +1 for the per-item Q load and epilogue
  assign_lpt(s->fwd, s->n_cta, [](const FwdItem& x) { return (int64_t)x.n_kv_tiles + 1; },
             s->fwd_cta_off);

  // ---- backward items ----
  std::vector<std::vector<int32_t>> seg_shards(n_segs);
  for (int i = 0; i < n_shards; ++i) seg_shards[s->shard_seg[i]].push_back(i);
  for (int g = 0; g < n_segs; ++g) {
    const int32_t kv0 = s->cu_k[g], kvl = s->cu_k[g + 1] - kv0;
    for (int32_t c0 = 0; c0 < kvl; c0 += FCP_TK) {
      BwdItem it;
      it.kv_row0 = kv0 + c0;
      it.kv_rows = std::min(FCP_TK, kvl - c0);
      it.kv_pos0 = c0;
      it.reserved = 0;
      it.sub_begin = (int32_t)s->bwd_sub.size();
      int32_t q_tiles = 0;
      for (int32_t i : seg_shards[g]) {
        const int32_t a = s->cu_q[i], len = s->cu_q[i + 1] - a, p = s->q_pos_off[i];
        if ((int64_t)p + len - 1 < c0 || len == 0) continue;     // no row of the shard sees the tile
        const int32_t t_first = std::max<int64_t>(0, (int64_t)c0 - p);
        const int32_t qt0 = t_first / FCP_BQ;
        BwdSub sb;
        sb.q_row0 = a + qt0 * FCP_BQ;
        sb.q_pos0 = p + qt0 * FCP_BQ;
        sb.q_rows = len - qt0 * FCP_BQ;
        sb.pad_row0 = s->shard_pad0[i] + qt0 * FCP_BQ;
        s->bwd_sub.push_back(sb);
        q_tiles += (sb.q_rows + FCP_BQ - 1) / FCP_BQ;
      }
      it.sub_end = (int32_t)s->bwd_sub.size();
      it.n_iters = q_tiles * s->G;
      // a KV tile no query sees still gets dk = dv = 0 written (n_iters == 0)
      for (int hk = 0; hk < s->Hkv; ++hk) {
        it.kv_head = hk;
        s->bwd.push_back(it);
        s->bwd_tile_pairs += it.n_iters;
      }
    }
  }
  stable_sort_desc(s->bwd, [](const BwdItem& x) { return (int64_t)x.n_iters; });
  // cost in inner iterations; +2 for the per-item K/V load and the dK/dV epilogue
  assign_lpt(s->bwd, s->n_cta, [](const BwdItem& x) { return (int64_t)x.n_iters + 2; },
             s->bwd_cta_off);

  // ---- workspace layout ----
  size_t o = 0;
  s->off_counters = o;  o = align_up(o + 256, 256);
  s->off_fwd = o;       o = align_up(o + s->fwd.size() * sizeof(FwdItem), 256);
  s->off_bwd = o;       o = align_up(o + s->bwd.size() * sizeof(BwdItem), 256);
  s->off_sub = o;       o = align_up(o + s->bwd_sub.size() * sizeof(BwdSub), 256);
  s->off_fwd_cta = o;   o = align_up(o + s->fwd_cta_off.size() * sizeof(int32_t), 256);
  s->off_bwd_cta = o;   o = align_up(o + s->bwd_cta_off.size() * sizeof(int32_t), 256);
  s->off_shard_meta = o;  // per padded 64-row tile: (local row0, valid rows)
  o = align_up(o + (size_t)(s->n_q_pad / FCP_BQ) * 2 * sizeof(int32_t), 256);
  s->off_lsed = o;      o = align_up(o + (size_t)s->Hq * s->n_q_pad * 2 * sizeof(float), 256);
  s->off_dq = o;        o = align_up(o + (size_t)s->n_q_pad * s->Hq * s->D * sizeof(float), 256);
  s->total = std::max<size_t>(o, 256);
  // host image of the list part of the workspace, uploaded with ONE copy (the per-rank host
  // latency matters on batches of short documents)
  s->image.assign(s->off_lsed, 0);
  auto put = [&](size_t off, const void* src, size_t bytes) {
    if (bytes) std::memcpy(s->image.data() + off, src, bytes);
  };
  put(s->off_fwd, s->fwd.data(), s->fwd.size() * sizeof(FwdItem));
  put(s->off_bwd, s->bwd.data(), s->bwd.size() * sizeof(BwdItem));
  put(s->off_sub, s->bwd_sub.data(), s->bwd_sub.size() * sizeof(BwdSub));
  put(s->off_fwd_cta, s->fwd_cta_off.data(), s->fwd_cta_off.size() * sizeof(int32_t));
  put(s->off_bwd_cta, s->bwd_cta_off.data(), s->bwd_cta_off.size() * sizeof(int32_t));
  put(s->off_shard_meta, s->tile_meta.data(), s->tile_meta.size() * sizeof(int32_t));
  *out = owner.release();
  return FCP_OK;
}

static int sched_create(const int32_t* cu_seqlens_q, const int32_t* q_pos_off,
                        const int32_t* shard_seg, int32_t n_shards, const int32_t* cu_seqlens_k,
                        int32_t n_segs, int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                        int32_t n_cta, fcp_sched** out) {
  return fcp_guard([&] {
    return sched_create_impl(cu_seqlens_q, q_pos_off, shard_seg, n_shards, cu_seqlens_k, n_segs,
                             n_q_heads, n_kv_heads, head_dim, n_cta, out);
  });
}

extern "C" int fcp_sched_create(const int32_t* cu_seqlens_q, const int32_t* q_pos_off,
                                const int32_t* shard_seg, int32_t n_shards,
                                const int32_t* cu_seqlens_k, int32_t n_segs, int32_t n_q_heads,
                                int32_t n_kv_heads, int32_t head_dim, fcp_sched** out) {
  return sched_create(cu_seqlens_q, q_pos_off, shard_seg, n_shards, cu_seqlens_k, n_segs,
                      n_q_heads, n_kv_heads, head_dim, fcp_sm_count(), out);
}

static int sched_from_plan(const fcp_plan* plan, int32_t rank, int32_t piece, int32_t n_q_heads,
                           int32_t n_kv_heads, int32_t head_dim, int32_t n_cta, fcp_sched** out) {
  RankView v;
  const int st = fcp_guard([&] { fcp_build_rank_view(*plan, rank, v, piece); return (int)FCP_OK; });
  if (st != FCP_OK) return st;
  return sched_create(v.cu_q.data(), v.q_pos_off.data(), v.shard_seg.data(),
                      (int32_t)v.q_pos_off.size(), v.cu_k.data(), (int32_t)v.kv_len.size(),
                      n_q_heads, n_kv_heads, head_dim, n_cta, out);
}

extern "C" int fcp_sched_from_plan(const fcp_plan* plan, int32_t rank, int32_t n_q_heads,
                                   int32_t n_kv_heads, int32_t head_dim, fcp_sched** out) {
  return fcp_sched_from_plan_piece(plan, rank, FCP_PIECE_FULL, n_q_heads, n_kv_heads, head_dim, out);
}

extern "C" int fcp_sched_from_plan_piece(const fcp_plan* plan, int32_t rank, int32_t piece,
                                         int32_t n_q_heads, int32_t n_kv_heads, int32_t head_dim,
                                         fcp_sched** out) {
  if (!plan || !out || rank < 0 || rank >= plan->n_ranks ||
      (piece != FCP_PIECE_FULL && piece != FCP_PIECE_LOCAL && piece != FCP_PIECE_PREFIX))
    return FCP_INVALID_ARG;
  return sched_from_plan(plan, rank, piece, n_q_heads, n_kv_heads, head_dim, fcp_sm_count(), out);
}

extern "C" void fcp_sched_destroy(fcp_sched* sched) { delete sched; }

extern "C" int fcp_sched_workspace_size(const fcp_sched* sched, size_t* device_bytes) {
  if (!sched || !device_bytes) return FCP_INVALID_ARG;
  *device_bytes = sched->total;
  return FCP_OK;
}

extern "C" int fcp_sched_get_info(const fcp_sched* sched, fcp_sched_info* out) {
  if (!sched || !out) return FCP_INVALID_ARG;
  out->n_fwd_items = (int32_t)sched->fwd.size();
  out->n_bwd_items = (int32_t)sched->bwd.size();
  out->fwd_kv_tiles = sched->fwd_kv_tiles;
  out->bwd_tile_pairs = sched->bwd_tile_pairs;
  out->useful_pairs = sched->useful_pairs;
  out->n_q = sched->n_q;
  out->n_kv = sched->n_kv;
  out->n_q_pad = sched->n_q_pad;
  return FCP_OK;
}

extern "C" int fcp_sched_get_list(const fcp_sched* sched, int32_t which, int32_t* out,
                                  int64_t cap_words, int64_t* n_words) {
  if (!sched || !n_words || cap_words < 0 || (cap_words > 0 && !out)) return FCP_INVALID_ARG;
  static_assert(sizeof(FwdItem) == 32 && sizeof(BwdItem) == 32 && sizeof(BwdSub) == 16, "layout");
  const void* src = nullptr;
  int64_t n = 0;
  switch (which) {
    case FCP_LIST_FWD_ITEMS: src = sched->fwd.data();         n = (int64_t)sched->fwd.size() * 8; break;
    case FCP_LIST_BWD_ITEMS: src = sched->bwd.data();         n = (int64_t)sched->bwd.size() * 8; break;
    case FCP_LIST_BWD_SUBS:  src = sched->bwd_sub.data();     n = (int64_t)sched->bwd_sub.size() * 4; break;
    case FCP_LIST_FWD_CTA:   src = sched->fwd_cta_off.data(); n = (int64_t)sched->fwd_cta_off.size(); break;
    case FCP_LIST_BWD_CTA:   src = sched->bwd_cta_off.data(); n = (int64_t)sched->bwd_cta_off.size(); break;
    default: return FCP_INVALID_ARG;
  }
  *n_words = n;
  const int64_t m = std::min(n, cap_words);
  if (m > 0) std::memcpy(out, src, (size_t)m * sizeof(int32_t));
  return FCP_OK;
}
