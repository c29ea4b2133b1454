// Host sharding planner: Algorithm 1 of FlashCP with the Whole-Doc /
// Per-Doc strategies of PAPER.md:62, 122-126, in the deterministic reading of DESIGN.md
// section 3.  Integer arithmetic only (64-bit loads, 128-bit ratio comparison).
#include <algorithm>
#include <cstring>
#include <memory>
#include <new>

#include "fcp_internal.h"

namespace {

struct Item { int32_t doc, start, len; };   // a movable Whole-Doc piece

struct Worker {
  int64_t tok = 0;
  uint64_t load = 0;
  std::vector<Item> items;
};

struct Pass {
  std::vector<Worker> w;
  std::vector<fcp_shard> chunks;   // Per-Doc chunks, fixed to their worker
  uint64_t max_load = 0, sum_load = 0;
};

// Worker with the smallest (load, index) among those for which `ok` holds.
template <class Pred>
int least_loaded(const std::vector<Worker>& w, Pred ok) {
  int best = -1;
  for (int j = 0; j < (int)w.size(); ++j)
    if (ok(w[j]) && (best < 0 || w[j].load < w[best].load)) best = j;
  return best;
}

// A = fcp_plan_opts.align_tokens (1 = Algorithm 1 proper; > 1 = the tile-aligned variant, fcp.h)
void run_pass(const std::vector<int32_t>& d, const std::vector<int32_t>& order, int k_per,
              int N, int64_t T, int32_t A, Pass& ps) {
  ps.w.assign(N, Worker());
  ps.chunks.clear();
  std::vector<Item> pool;
  // Per-Doc: 2N chunks, chunk c and 2N-1-c on worker c; d mod 2N tokens at the
  // head of the document become an ordinary Whole-Doc item.
  // With A > 1 the chunk length is a multiple of A, the head item is the aligned part of the
  // leftover and its ragged rest (< A tokens) is a movable item at the document's end that
  // starts on the worker of the last chunk.
  for (int x = 0; x < k_per; ++x) {
    const int32_t i = order[x];
    const int32_t q = (int32_t)(d[i] / (2 * (int64_t)N * A) * A);
    if (q == 0) {
      pool.push_back({i, 0, d[i]});
      continue;
    }
    const int32_t r = (d[i] - 2 * N * q) / A * A, e = d[i] - 2 * N * q - r;
    if (r > 0) pool.push_back({i, 0, r});
    for (int c = 0; c < 2 * N; ++c) {
      const int j = c < N ? c : 2 * N - 1 - c;
      ps.chunks.push_back({i, r + c * q, q, j});
      ps.w[j].tok += q;
      ps.w[j].load += fcp_W(r + c * q, q);
    }
    if (e > 0) {
      ps.w[0].items.push_back({i, d[i] - e, e});
      ps.w[0].tok += e;
      ps.w[0].load += fcp_W(d[i] - e, e);
    }
  }
  for (size_t x = k_per; x < order.size(); ++x) pool.push_back({order[x], 0, d[order[x]]});
  std::stable_sort(pool.begin(), pool.end(), [](const Item& a, const Item& b) {
    return a.len != b.len ? a.len > b.len : a.doc < b.doc;
  });
  // Lines 5-9: longest first onto the least-loaded worker (by attention workload).
  for (const Item& it : pool) {
    Worker& t = ps.w[least_loaded(ps.w, [](const Worker&) { return true; })];
    t.items.push_back(it);
    t.tok += it.len;
    t.load += fcp_W(it.start, it.len);
  }
  // Lines 10-16: enforce Eq. 2 by Whole-Doc sharding.  The donor is the worker with the most
  // tokens; it gives away whole items that fit, else the head of its longest item.
  for (;;) {
    int a = 0;
    for (int j = 1; j < N; ++j)
      if (ps.w[j].tok > ps.w[a].tok) a = j;
    if (ps.w[a].tok == T) break;
    int64_t excess = ps.w[a].tok - T;
    while (excess > 0) {
      const int b = least_loaded(ps.w, [T](const Worker& x) { return x.tok < T; });
      const int64_t room = std::min<int64_t>(excess, T - ps.w[b].tok);
      std::vector<Item>& src = ps.w[a].items;
      int pick = -1;
      for (int x = 0; x < (int)src.size(); ++x)       // smallest whole item that fits
        if (src[x].len <= room &&
            (pick < 0 || src[x].len < src[pick].len ||
             (src[x].len == src[pick].len && src[x].doc < src[pick].doc)))
          pick = x;
      Item moved;
      if (pick >= 0) {
        moved = src[pick];
        src.erase(src.begin() + pick);
      } else {
        // cut the head of the longest item (A > 1: of the longest item that starts on a multiple
        // of A, and a multiple of A tokens; a hand-over below A comes from the shortest item)
        int32_t g = (int32_t)room;
        const bool ragged = g < A;
        bool on_grid = false;
        for (int x = 0; x < (int)src.size() && !ragged; ++x) on_grid |= src[x].start % A == 0;
        for (int x = 0; x < (int)src.size(); ++x) {
          if (on_grid && src[x].start % A != 0) continue;
          const bool better = ragged ? src[x].len < src[pick < 0 ? x : pick].len
                                     : src[x].len > src[pick < 0 ? x : pick].len;
          if (pick < 0 || better || (src[x].len == src[pick].len && src[x].doc < src[pick].doc))
            pick = x;
        }
        if (on_grid) g = g / A * A;
        moved = {src[pick].doc, src[pick].start, g};
        src[pick].start += g;
        src[pick].len -= g;
      }
      const uint64_t wl = fcp_W(moved.start, moved.len);
      ps.w[a].tok -= moved.len;  ps.w[a].load -= wl;
      ps.w[b].tok += moved.len;  ps.w[b].load += wl;
      ps.w[b].items.push_back(moved);
      excess -= moved.len;
    }
  }
  ps.max_load = ps.sum_load = 0;
  for (const Worker& x : ps.w) {
    ps.max_load = std::max(ps.max_load, x.load);
    ps.sum_load += x.load;
  }
}

}  // namespace

extern "C" int fcp_plan_create(const int32_t* doc_lengths, int32_t n_docs, int32_t n_ranks,
                               const fcp_plan_opts* opts, fcp_plan** out) {
  if (!doc_lengths || !out || n_docs < 1 || n_ranks < 1) return FCP_INVALID_ARG;
  int64_t r_ppm = 1050000;
  int32_t strategy = FCP_STRATEGY_HYBRID, align = 1;
  if (opts) {
    if (opts->align_tokens < 0) return FCP_INVALID_ARG;
    if (opts->align_tokens > 1) align = opts->align_tokens;
    if (opts->imbalance_ppm != 0) r_ppm = opts->imbalance_ppm;
    strategy = opts->strategy;
  }
  if (r_ppm < 1000000) return FCP_INVALID_ARG;
  if (strategy < 0 || strategy > FCP_STRATEGY_PER_SEQ) return FCP_UNSUPPORTED;
  int64_t C = 0;
  for (int i = 0; i < n_docs; ++i) {
    if (doc_lengths[i] < 1) return FCP_INVALID_ARG;
    C += doc_lengths[i];
  }
  if (C % n_ranks != 0 || C > INT32_MAX) return FCP_INVALID_ARG;
  if (strategy == FCP_STRATEGY_PER_SEQ && C % (2 * (int64_t)n_ranks) != 0) return FCP_INVALID_ARG;
  const int N = n_ranks;
  const int64_t T = C / N;
  return fcp_guard([&]() -> int {
  std::unique_ptr<fcp_plan> p(new fcp_plan());
  p->d.assign(doc_lengths, doc_lengths + n_docs);
  p->off.resize(n_docs + 1);
  p->off[0] = 0;
  for (int i = 0; i < n_docs; ++i) p->off[i + 1] = p->off[i] + p->d[i];
  p->n_ranks = N;  p->C = C;  p->T = T;

  std::vector<fcp_shard> all;
  if (strategy == FCP_STRATEGY_PER_SEQ) {
    // Llama3 CP baseline: the packed sequence in 2N equal chunks regardless of
    // document borders, chunks c and 2N-1-c on worker c; one shard per document piece.
    const int64_t q = C / (2 * N);
    int k = 0;
    for (int c = 0; c < 2 * N; ++c) {
      const int j = c < N ? c : 2 * N - 1 - c;
      const int64_t lo = (int64_t)c * q, hi = lo + q;
      while (p->off[k + 1] <= lo) ++k;
      for (int kk = k; kk < n_docs && p->off[kk] < hi; ++kk) {
        const int64_t a = std::max(lo, p->off[kk]), b = std::min(hi, p->off[kk + 1]);
        if (a < b) all.push_back({kk, (int32_t)(a - p->off[kk]), (int32_t)(b - a), j});
      }
    }
    p->n_passes = 1;
  }

  std::vector<int32_t> order(n_docs);
  for (int i = 0; i < n_docs; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(),
                   [&](int32_t a, int32_t b) { return p->d[a] > p->d[b]; });   // line 1

  int k_per = strategy == FCP_STRATEGY_ALL_PER_DOC ? n_docs : 0;
  const int k_last = strategy == FCP_STRATEGY_WHOLE_DOC ? 0 : n_docs;
  Pass ps;
  for (; strategy != FCP_STRATEGY_PER_SEQ;) {          // line 4
    run_pass(p->d, order, k_per, N, T, align, ps);
    ++p->n_passes;
    // Cur_R > R  <=>  max * N * 1e6 > R_ppm * sum, in 128 bits
    const unsigned __int128 lhs = (unsigned __int128)ps.max_load * (uint64_t)N * 1000000u;
    const unsigned __int128 rhs = (unsigned __int128)ps.sum_load * (uint64_t)r_ppm;
    if (!(lhs > rhs) || k_per >= k_last) break;
    ++k_per;                                           // lines 19-23
  }
  if (strategy != FCP_STRATEGY_PER_SEQ) {
    p->per_doc.assign(order.begin(), order.begin() + k_per);
    p->max_load = ps.max_load;
    p->sum_load = ps.sum_load;
    all = ps.chunks;
    for (int j = 0; j < N; ++j)
      for (const Item& it : ps.w[j].items) all.push_back({it.doc, it.start, it.len, j});
  } else {
    std::vector<uint64_t> load(N, 0);
    for (const fcp_shard& s : all) load[s.rank] += fcp_W(s.start, s.len);
    for (uint64_t x : load) {
      p->max_load = std::max(p->max_load, x);
      p->sum_load += x;
    }
  }
  std::sort(all.begin(), all.end(), [](const fcp_shard& a, const fcp_shard& b) {
    if (a.rank != b.rank) return a.rank < b.rank;
    if (a.doc != b.doc) return a.doc < b.doc;
    return a.start < b.start;
  });
  for (const fcp_shard& s : all) {
    if (!p->shards.empty()) {
      fcp_shard& l = p->shards.back();
      if (l.rank == s.rank && l.doc == s.doc && l.start + l.len == s.start) {
        l.len += s.len;
        continue;
      }
    }
    p->shards.push_back(s);
  }
  p->rank_begin.assign(N + 1, 0);
  for (const fcp_shard& s : p->shards) ++p->rank_begin[s.rank + 1];
  for (int j = 0; j < N; ++j) p->rank_begin[j + 1] += p->rank_begin[j];
  *out = p.release();
  return FCP_OK;
  });
}

extern "C" void fcp_plan_destroy(fcp_plan* plan) { delete plan; }

extern "C" int fcp_plan_shards(const fcp_plan* plan, int32_t rank, fcp_shard* out, int32_t cap,
                               int32_t* n_out) {
  if (!plan || !n_out || cap < 0 || rank < -1 || rank >= plan->n_ranks) return FCP_INVALID_ARG;
  const int32_t b = rank < 0 ? 0 : plan->rank_begin[rank];
  const int32_t e = rank < 0 ? (int32_t)plan->shards.size() : plan->rank_begin[rank + 1];
  *n_out = e - b;
  const int32_t n = std::min(cap, e - b);
  if (n > 0) {
    if (!out) return FCP_INVALID_ARG;
    std::memcpy(out, plan->shards.data() + b, sizeof(fcp_shard) * n);
  }
  return e - b > cap ? FCP_BUFFER_TOO_SMALL : FCP_OK;
}

extern "C" int fcp_plan_perdoc(const fcp_plan* plan, int32_t* doc_ids, int32_t cap,
                               int32_t* n_out) {
  if (!plan || !n_out || cap < 0) return FCP_INVALID_ARG;
  const int32_t cnt = (int32_t)plan->per_doc.size();
  *n_out = cnt;
  const int32_t n = std::min(cap, cnt);
  if (n > 0) {
    if (!doc_ids) return FCP_INVALID_ARG;
    std::memcpy(doc_ids, plan->per_doc.data(), sizeof(int32_t) * n);
  }
  return cnt > cap ? FCP_BUFFER_TOO_SMALL : FCP_OK;
}

void fcp_build_rank_view(const fcp_plan& p, int32_t rank, RankView& v, int32_t piece) {
  const int n = (int)p.d.size();
  std::vector<int32_t> E(n, 0), seg_of(n, -1);
  const int32_t b = p.rank_begin[rank], e = p.rank_begin[rank + 1];
  for (int32_t i = b; i < e; ++i)
    E[p.shards[i].doc] = std::max(E[p.shards[i].doc], p.shards[i].start + p.shards[i].len);
  v = RankView();
  v.cu_k.push_back(0);
  for (int k = 0; k < n; ++k)
    if (E[k] > 0) {
      seg_of[k] = (int32_t)v.kv_len.size();
      v.kv_src_start.push_back((int32_t)p.off[k]);
      v.kv_len.push_back(E[k]);
      v.seg_doc.push_back(k);
      v.cu_k.push_back(v.cu_k.back() + E[k]);
    }
  v.n_kv = v.cu_k.back();
  v.cu_q.push_back(0);
  int64_t own_in_prefix = 0;
  for (int32_t i = b; i < e; ++i) {
    const fcp_shard& s = p.shards[i];
    v.cu_q.push_back(v.cu_q.back() + s.len);
    v.q_pos_off.push_back(s.start);
    v.shard_seg.push_back(seg_of[s.doc]);
    v.load += fcp_W(s.start, s.len);
    if (s.start + s.len != p.d[s.doc]) v.nonlast += s.len;   // S-hat
    own_in_prefix += s.len;        // every shard lies inside [0, E) of its document
  }
  v.n_q = v.cu_q.back();
  v.remote = v.n_kv - own_in_prefix;
  if (piece == FCP_PIECE_FULL) return;
  // Local / prefix split (fcp.h section 2b): one KV segment per shard.  LOCAL = the shard's own
  // tokens [p, p+s), causal from its first key; PREFIX = the tokens [0, p) before it, all
  // visible.  The distinct remote tokens of PREFIX are those of the unsplit gather.
  v.cu_k.assign(1, 0);
  v.kv_src_start.clear();
  v.kv_len.clear();
  v.seg_doc.clear();
  for (int32_t i = b; i < e; ++i) {
    const fcp_shard& s = p.shards[i];
    const bool local = piece == FCP_PIECE_LOCAL;
    v.q_pos_off[i - b] = local ? 0 : s.start;
    v.shard_seg[i - b] = i - b;
    v.kv_src_start.push_back((int32_t)(p.off[s.doc] + (local ? s.start : 0)));
    v.kv_len.push_back(local ? s.len : s.start);
    v.seg_doc.push_back(s.doc);
    v.cu_k.push_back(v.cu_k.back() + v.kv_len.back());
  }
  v.n_kv = v.cu_k.back();
  if (piece == FCP_PIECE_LOCAL) v.remote = 0;
}

static bool valid_piece(int32_t piece) {
  return piece == FCP_PIECE_FULL || piece == FCP_PIECE_LOCAL || piece == FCP_PIECE_PREFIX;
}

extern "C" int fcp_plan_rank_stats(const fcp_plan* plan, int32_t rank, fcp_rank_stats* out) {
  return fcp_plan_piece_stats(plan, rank, FCP_PIECE_FULL, out);
}

extern "C" int fcp_plan_piece_stats(const fcp_plan* plan, int32_t rank, int32_t piece,
                                    fcp_rank_stats* out) {
  if (!plan || !out || rank < 0 || rank >= plan->n_ranks || !valid_piece(piece))
    return FCP_INVALID_ARG;
  RankView v;
  const int st = fcp_guard([&] { fcp_build_rank_view(*plan, rank, v, piece); return (int)FCP_OK; });
  if (st != FCP_OK) return st;
  out->n_shards = (int32_t)v.q_pos_off.size();
  out->n_segs = (int32_t)v.kv_len.size();
  out->n_q = v.n_q;
  out->n_kv = v.n_kv;
  out->remote_tokens = v.remote;
  out->nonlast_tokens = v.nonlast;
  out->load = v.load;
  return FCP_OK;
}

extern "C" int fcp_plan_stats(const fcp_plan* plan, fcp_stats* out) {
  if (!plan || !out) return FCP_INVALID_ARG;
  std::memset(out, 0, sizeof(*out));
  const int N = plan->n_ranks;
  out->n_ranks = N;
  out->n_docs = (int32_t)plan->d.size();
  out->n_shards = (int32_t)plan->shards.size();
  out->n_per_doc = (int32_t)plan->per_doc.size();
  out->n_passes = plan->n_passes;
  out->context_len = plan->C;
  out->tokens_per_rank = plan->T;
  out->max_load = plan->max_load;
  out->sum_load = plan->sum_load;
  out->imbalance_ppm =
      (int64_t)((unsigned __int128)plan->max_load * (uint64_t)N * 1000000u / plan->sum_load);
  out->eq4_tokens = plan->T * (N - 1);                         // Eq. 4
  int64_t max_nonlast = 0;
  for (int r = 0; r < N; ++r) {
    RankView v;
    const int st = fcp_guard([&] { fcp_build_rank_view(*plan, r, v); return (int)FCP_OK; });
    if (st != FCP_OK) return st;
    max_nonlast = std::max(max_nonlast, v.nonlast);
    out->max_remote_tokens = std::max(out->max_remote_tokens, v.remote);
    out->sum_remote_tokens += v.remote;
    out->max_gathered_tokens = std::max(out->max_gathered_tokens, v.n_kv);
    out->sum_gathered_tokens += v.n_kv;
  }
  out->eq5_tokens = (int64_t)(N - 1) * max_nonlast;            // Eq. 5
  return FCP_OK;
}

extern "C" int fcp_rank_layout(const fcp_plan* plan, int32_t rank, fcp_layout* out) {
  return fcp_piece_layout(plan, rank, FCP_PIECE_FULL, out);
}

extern "C" int fcp_piece_layout(const fcp_plan* plan, int32_t rank, int32_t piece,
                                fcp_layout* out) {
  if (!plan || !out || rank < 0 || rank >= plan->n_ranks || !valid_piece(piece))
    return FCP_INVALID_ARG;
  RankView v;
  const int st = fcp_guard([&] { fcp_build_rank_view(*plan, rank, v, piece); return (int)FCP_OK; });
  if (st != FCP_OK) return st;
  auto put = [](int32_t* dst, const std::vector<int32_t>& src) {
    if (dst && !src.empty()) std::memcpy(dst, src.data(), sizeof(int32_t) * src.size());
  };
  put(out->cu_seqlens_q, v.cu_q);
  put(out->q_pos_off, v.q_pos_off);
  put(out->shard_seg, v.shard_seg);
  put(out->cu_seqlens_k, v.cu_k);
  put(out->kv_src_start, v.kv_src_start);
  put(out->kv_len, v.kv_len);
  if (out->q_token_index) {
    int64_t w = 0;
    for (int32_t i = plan->rank_begin[rank]; i < plan->rank_begin[rank + 1]; ++i) {
      const fcp_shard& s = plan->shards[i];
      for (int32_t t = 0; t < s.len; ++t)
        out->q_token_index[w++] = (int32_t)(plan->off[s.doc] + s.start + t);
    }
  }
  if (out->kv_token_index) {
    int64_t w = 0;
    for (size_t g = 0; g < v.kv_len.size(); ++g)
      for (int32_t t = 0; t < v.kv_len[g]; ++t) out->kv_token_index[w++] = v.kv_src_start[g] + t;
  }
  return FCP_OK;
}

extern "C" const char* fcp_strerror(int status) {
  switch (status) {
    case FCP_OK: return "ok";
    case FCP_INVALID_ARG: return "invalid argument";
    case FCP_UNSUPPORTED: return "unsupported configuration";
    case FCP_BUFFER_TOO_SMALL: return "buffer too small";
    case FCP_CUDA: return "CUDA error";
    case FCP_MISALIGNED: return "misaligned pointer";
    case FCP_NO_MEMORY: return "out of host memory";
    case FCP_TOO_LARGE: return "schedule workspace larger than FCP_STATIC_WORKSPACE_BYTES";
    default: return "unknown status";
  }
}

extern "C" const char* fcp_version(void) { return "sm_100a;fcp-0.2"; }
