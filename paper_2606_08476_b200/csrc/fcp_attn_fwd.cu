// Document-masked causal attention forward for sm_100a.
//
// One persistent CTA per SM.  A work item is one 128-row q tile of one shard for a pack of NQ
// query heads that share a kv head (GQA): the NQ tiles share every K/V tile staged in shared
// memory and ping-pong on the tensor core — while the softmax warps of one tile work, the
// MMAs of the other tile run.
//
//   warp 0      TMA producer   Q (once per item), K/V tiles through a ring of smem stages
//   warp 1      MMA issuer     one elected thread: S_t = Q_t K^T (SS), O_t += P_t V (A = P from
//                              TMEM, B = V MN-major); it probes the next group's barriers before
//                              the last MMAs of the current group (the tcgen05 queue is ~5 deep)
//   warps 4..   softmax        one warpgroup per q tile, one query row per thread: mask from
//                              (q_pos0 + row, kv_len), online softmax in the log2 domain whose
//                              fast path exponentiates against the running max of the earlier
//                              tiles (no max -> exp dependency) and rescales O only when a row
//                              grew by more than 2^8; P written back to TMEM as bf16 over S,
//                              epilogue o = O / l
//
// TMEM columns: S_t at 128 t, O_t at 128 (NQ + t); P_t aliases the first 64 columns of S_t.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "fcp_internal.h"
#include "fcp_sm100.cuh"
#include "fcp_tma.h"

#ifdef FCP_EXP_TRACE
__device__ long long g_trace_fwd[64 * 16];
extern "C" int fcp_debug_trace_fwd(long long* out) {
  return (int)cudaMemcpyFromSymbol(out, g_trace_fwd, sizeof(g_trace_fwd));
}
#define FTRACE(n, id)                                                                  \
  do {                                                                                 \
    if (blockIdx.x == 0 && (n) >= 50u && (n) < 114u && (threadIdx.x & 31) == 0)        \
      g_trace_fwd[((n) - 50u) * 16 + (id)] = clock64();                                \
  } while (0)
#else
#define FTRACE(n, id)
#endif

namespace {
using namespace fcp;

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.0f;   // log2 units: rescale O only when the max grew by > 2^8

template <int D, int NQ>
struct FwdCfg {
  static constexpr int kTileBytes = 128 * D * 2;           // one Q, K or V tile
  static constexpr int kPanelBytes = 128 * 128;            // 128 rows x 64 bf16
  static constexpr int kPanels = D / 64;
  static constexpr int kStages = (D == 128) ? 4 : 6;       // ring slots, each one K or V tile
  // softmax warpgroups per q tile: each takes 128 / kHalves key columns of every KV tile.
  // MUFU (16 ex2/clk/SM) bounds the softmax of a 128x128 tile at 1024 clocks whatever the warp
  // count, so one warpgroup per tile (no cross-warpgroup exchange) is the faster layout.
  static constexpr int kHalves = 1;
  static constexpr int kSoftmaxThreads = 128 * kHalves;    // per q tile
  static constexpr int kThreads = 128 + kSoftmaxThreads * NQ;
  static constexpr int kTmemCols = 256 * NQ;
  static constexpr int kSmemData = (NQ + kStages) * kTileBytes;
  static constexpr int kXchBytes = NQ * 2 * 128 * 4;       // row max / row sum exchange (kHalves = 2)
  static constexpr int kSmemBytes = 1024 + kSmemData + kXchBytes + 1024;
  // registers per thread after setmaxnreg (multiples of 8).  The CTA owns (launch registers x
  // threads): the sum over its warpgroups must stay below.
  static constexpr int kLaunchRegs = (65536 / kThreads) / 8 * 8 > 255 ? 248 : (65536 / kThreads) / 8 * 8;
  static constexpr int kRegsCtl = 80;
  static constexpr int kRegsSoftmaxRaw =
      (kLaunchRegs * (kThreads / 128) - kRegsCtl) / (kHalves * NQ) / 8 * 8;
  static constexpr int kRegsSoftmax = kRegsSoftmaxRaw > 232 ? 232 : kRegsSoftmaxRaw;
  static constexpr int kTail = 3;   // MMAs issued after the probe of the next group's barriers
};

struct FwdBarriers {
  uint64_t q_full, q_empty;
  uint64_t kv_full[8], kv_empty[8];
  uint64_t s_full[2], p_ready[2], o_full[2], o_empty[2];
  uint32_t tmem_base;
};

template <int D, int NQ>
__global__ void __launch_bounds__(FwdCfg<D, NQ>::kThreads, 1)
fcp_attn_fwd_kernel(const __grid_constant__ CUtensorMap tmap_q,
                    const __grid_constant__ CUtensorMap tmap_k,
                    const __grid_constant__ CUtensorMap tmap_v,
                    const FwdItem* __restrict__ items, const int32_t* __restrict__ cta_off,
                    __nv_bfloat16* __restrict__ o, float* __restrict__ lse,
                    int64_t n_q, int Hq, float scale_log2) {
  using Cfg = FwdCfg<D, NQ>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) &
                                             ~uintptr_t(1023));
  uint8_t* q_smem = smem;                                  // NQ tiles
  uint8_t* ring = smem + NQ * Cfg::kTileBytes;             // kStages tiles
  float* xch = reinterpret_cast<float*>(smem + Cfg::kSmemData);   // [NQ][2 halves][128 rows]
  FwdBarriers* bars = reinterpret_cast<FwdBarriers*>(smem + Cfg::kSmemData + Cfg::kXchBytes);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    mbar_init(&bars->q_full, 1);
    mbar_init(&bars->q_empty, 1);
    for (int i = 0; i < Cfg::kStages; ++i) {
      mbar_init(&bars->kv_full[i], 1);
      mbar_init(&bars->kv_empty[i], 1);
    }
    for (int t = 0; t < NQ; ++t) {
      mbar_init(&bars->s_full[t], 1);
      mbar_init(&bars->p_ready[t], Cfg::kSoftmaxThreads);
      mbar_init(&bars->o_full[t], 1);
      mbar_init(&bars->o_empty[t], Cfg::kSoftmaxThreads);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<Cfg::kTmemCols>(&bars->tmem_base);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;
  const int item_begin = cta_off[blockIdx.x], item_end = cta_off[blockIdx.x + 1];   // this CTA's work list

  if (warp < 4) {
    reg_dealloc<Cfg::kRegsCtl>();
    if (warp == 0 && lane == 0) {
      // ---------------------------------------------------------------- TMA producer
      prefetch_tmap(&tmap_q);
      prefetch_tmap(&tmap_k);
      prefetch_tmap(&tmap_v);
      uint32_t kv_n = 0, item_n = 0;
      for (int idx = item_begin; idx < item_end; ++idx) {
        const FwdItem it = items[idx];
        if (it.n_kv_tiles == 0) continue;
        mbar_wait(&bars->q_empty, (item_n & 1) ^ 1);
        mbar_arrive_expect_tx(&bars->q_full, NQ * Cfg::kTileBytes);
        for (int t = 0; t < NQ; ++t)
          for (int pn = 0; pn < Cfg::kPanels; ++pn)
            tma_load_3d(q_smem + t * Cfg::kTileBytes + pn * Cfg::kPanelBytes, &tmap_q,
                        &bars->q_full, pn * 64, it.head0 + t, it.q_row0);
        for (int j = 0; j < it.n_kv_tiles; ++j) {
          for (int which = 0; which < 2; ++which) {
            const uint32_t slot = kv_n % Cfg::kStages, ph = (kv_n / Cfg::kStages) & 1;
            mbar_wait(&bars->kv_empty[slot], ph ^ 1);
            mbar_arrive_expect_tx(&bars->kv_full[slot], Cfg::kTileBytes);
            for (int pn = 0; pn < Cfg::kPanels; ++pn)
              tma_load_3d(ring + slot * Cfg::kTileBytes + pn * Cfg::kPanelBytes,
                          which == 0 ? &tmap_k : &tmap_v, &bars->kv_full[slot], pn * 64,
                          it.kv_head, it.kv_row0 + j * FCP_TK);
            ++kv_n;
          }
        }
        ++item_n;
      }
    } else if (warp == 1 && elect_one()) {
      // ---------------------------------------------------------------- MMA issuer
      // One elected thread.  Per KV tile j and q tile t one group: O_t += P_t(j) V_j, then
      // S_t = Q_t K_{j+1}^T.  The barriers of the next group are probed (non-blocking) before the
      // last kTail MMAs of the current group so the ~5-deep tcgen05 queue never drains while
      // this thread looks at a barrier; descriptors are 32-bit adds on precomputed low words.
      constexpr uint32_t idesc_qk = umma_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = umma_idesc_bf16(128, D, 0, 1);
      constexpr int kTail = Cfg::kTail;
      constexpr int kSteps = D / 16;
      constexpr uint32_t kHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO, version, swizzle
      constexpr uint32_t kTileStep = Cfg::kTileBytes >> 4;
      auto lo_word = [](uint32_t saddr, uint32_t lbo) { return ((saddr & 0x3FFFF) >> 4) | ((lbo >> 4) << 16); };
      auto desc = [](uint32_t lo) { return ((uint64_t)kHi << 32) | lo; };
      const uint32_t q_kmaj = lo_word(smem_u32(q_smem), 16);                     // A of S (tile 0)
      const uint32_t ring_kmaj = lo_word(smem_u32(ring), 16);                    // K tile, slot 0
      const uint32_t ring_mnmaj = lo_word(smem_u32(ring), Cfg::kPanelBytes);     // V tile, slot 0

      auto issue_qk = [&](int t, uint32_t kslot, int kk0, int kk1) {
        const uint32_t a0 = q_kmaj + t * kTileStep, b0 = ring_kmaj + kslot * kTileStep;
#pragma unroll
        for (int kk = kk0; kk < kk1; ++kk) {
          const uint32_t off = ((kk >> 2) * Cfg::kPanelBytes + (kk & 3) * 32) >> 4;
          umma_ss(tmem_base + t * 128, desc(a0 + off), desc(b0 + off), idesc_qk, kk > 0);
        }
      };
      auto issue_pv = [&](int t, uint32_t vslot, bool acc, int kk0, int kk1) {
        const uint32_t b0 = ring_mnmaj + vslot * kTileStep;
#pragma unroll
        for (int kk = kk0; kk < kk1; ++kk)
          umma_ts(tmem_base + (NQ + t) * 128, tmem_base + t * 128 + kk * 8,
                  desc(b0 + kk * (2048 >> 4)), idesc_pv, (acc || kk > 0) ? 1u : 0u);
      };
      auto ring_next = [](uint32_t& s_, uint32_t& p_) {
        if (++s_ == (uint32_t)Cfg::kStages) { s_ = 0; p_ ^= 1; }
      };

      uint32_t slot = 0, sph = 0;      // ring position / phase parity of the next tile to consume
      uint32_t pp[NQ];                 // parity of the next p_ready phase of each q tile
#pragma unroll
      for (int t = 0; t < NQ; ++t) pp[t] = 0;
      uint32_t iph = 0;                // item parity (q_full / o_empty / o_full)
#ifdef FCP_EXP_TRACE
      uint32_t tn = 0;
#endif

      for (int idx = item_begin; idx < item_end; ++idx) {
        const int n = items[idx].n_kv_tiles;
        if (n == 0) continue;
        mbar_wait(&bars->q_full, iph);
        mbar_wait(&bars->kv_full[slot], sph);
        tc_fence_after();
#pragma unroll
        for (int t = 0; t < NQ; ++t) {
          issue_qk(t, slot, 0, kSteps);
          umma_commit(&bars->s_full[t]);
        }
        umma_commit(&bars->kv_empty[slot]);
        if (n == 1) umma_commit(&bars->q_empty);
        ring_next(slot, sph);
        bool ok = false;               // barriers of the upcoming group already seen complete
        for (int j = 0; j < n; ++j) {
          const bool has_next = j + 1 < n;
          const uint32_t vslot = slot, vph = sph;
          uint32_t kslot = slot, kph = sph;
          ring_next(kslot, kph);
#pragma unroll
          for (int t = 0; t < NQ; ++t) {
            FTRACE(tn, 8 + 3 * t);
            if (!ok) {
              mbar_wait(&bars->p_ready[t], pp[t]);
              if (j == 0) mbar_wait(&bars->o_empty[t], iph ^ 1);
              if (t == 0) {
                mbar_wait(&bars->kv_full[vslot], vph);
                if (has_next) mbar_wait(&bars->kv_full[kslot], kph);
              }
            }
            FTRACE(tn, 9 + 3 * t);
            pp[t] ^= 1;
            tc_fence_after();
            // probe of the next group: (t+1, j), else (0, j+1), else none (next item: blocking)
            auto probe_next = [&]() -> bool {
              if (t + 1 < NQ) {
                const int t1 = (t + 1 < NQ) ? t + 1 : 0;
                return mbar_test(&bars->p_ready[t1], pp[t1]) &
                       (j > 0 || mbar_test(&bars->o_empty[t1], iph ^ 1));
              }
              if (!has_next) return false;
              uint32_t v1 = kslot, v1p = kph;
              ring_next(v1, v1p);                  // V_{j+1}
              uint32_t k2 = v1, k2p = v1p;
              ring_next(k2, k2p);                  // K_{j+2}
              return mbar_test(&bars->p_ready[0], pp[0]) & mbar_test(&bars->kv_full[v1], v1p) &
                     (j + 2 >= n || mbar_test(&bars->kv_full[k2], k2p));
            };
            if (has_next) {
              issue_pv(t, vslot, j > 0, 0, 8);
              issue_qk(t, kslot, 0, kSteps - kTail);
              ok = probe_next();
              issue_qk(t, kslot, kSteps - kTail, kSteps);
              umma_commit(&bars->s_full[t]);
            } else {
              issue_pv(t, vslot, j > 0, 0, 8 - kTail);
              ok = probe_next();
              issue_pv(t, vslot, true, 8 - kTail, 8);
              umma_commit(&bars->o_full[t]);
            }
            FTRACE(tn, 10 + 3 * t);
          }
          umma_commit(&bars->kv_empty[vslot]);
          ring_next(slot, sph);
          if (has_next) {
            umma_commit(&bars->kv_empty[kslot]);
            ring_next(slot, sph);
            if (j + 2 == n) umma_commit(&bars->q_empty);
          }
#ifdef FCP_EXP_TRACE
          ++tn;
#endif
        }
        iph ^= 1;
      }
    }
  } else {
    // ------------------------------------------------------------------ softmax + epilogue
    // kHalves warpgroups per q tile, each taking 128 / kHalves key columns of every KV tile (a
    // warp reaches TMEM lanes 32*(warp%4)..+31 only, so each warpgroup covers all 128 query
    // rows).  One query row per thread.  Online softmax in the log2 domain:
    //   fast path  p = exp2(s c - m) with the running max m of the earlier tiles while the tile
    //              max is computed on the side (no max -> exp dependency); valid as long as no
    //              row of the warp exceeds m by more than 2^kRescaleThreshold;
    //   exact path (first tile of a row, or a row that grew): tile max first, m and O rescaled.
    constexpr int kH = Cfg::kHalves;
    constexpr int kCW = 128 / kH;                  // key columns per thread and KV tile
    constexpr int kOW = D / kH;                    // O columns per thread in rescale / epilogue
    reg_alloc<Cfg::kRegsSoftmax>();
    const int t = (warp - 4) / (4 * kH);           // q tile of this warp
    const int half = ((warp - 4) >> 2) % kH;       // key-column part
    const int row = (warp & 3) * 32 + lane;        // query row = TMEM lane
    const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem_base + lane_addr + t * 128;
    const uint32_t tP = tS + half * (kCW / 2);     // bf16 P of this thread's columns
    const uint32_t tO = tmem_base + lane_addr + (NQ + t) * 128 + half * kOW;
    float* xch_mine = xch + (t * 2 + half) * 128 + row;
    const float* xch_other = xch + (t * 2 + (half ^ 1)) * 128 + row;
    const uint32_t pair_bar = 1 + t;               // named barrier of the tile's warpgroups (kH = 2)
    uint32_t s_ph = 0, o_ph = 0;
#ifdef FCP_EXP_TRACE
    uint32_t tn = 0;
#endif

    for (int idx = item_begin; idx < item_end; ++idx) {
      const FwdItem it = items[idx];
      const int n = it.n_kv_tiles;
      const int head = it.head0 + t;
      const bool row_valid = row < it.q_rows;
      __nv_bfloat16* o_row = o + ((int64_t)(it.q_row0 + row) * Hq + head) * D + half * kOW;
      float* lse_row = lse + (int64_t)head * n_q + it.q_row0 + row;
      if (n == 0) {                                 // no visible key: o = 0, lse = -inf
        if (row_valid) {
          for (int c = 0; c < kOW; c += 8) *reinterpret_cast<int4*>(o_row + c) = make_int4(0, 0, 0, 0);
          if (half == 0) *lse_row = -INFINITY;
        }
        continue;
      }
      // last visible key (segment position) of this row; may be negative
      const int limit = min(it.q_pos0 + row, it.kv_len - 1);
      const int warp_min_limit = min(it.q_pos0 + (warp & 3) * 32, it.kv_len - 1);
      float m = -INFINITY, l = 0.f;

      for (int j = 0; j < n; ++j) {
        if ((warp & (4 * kH - 1)) == 0) FTRACE(tn, 4 * t);
        mbar_wait(&bars->s_full[t], s_ph);
        if ((warp & (4 * kH - 1)) == 0) FTRACE(tn, 4 * t + 1);
        s_ph ^= 1;
        tc_fence_after();
        uint32_t sr[kCW / 32][32];
#pragma unroll
        for (int c = 0; c < kCW / 32; ++c) tmem_ld32(tS + half * kCW + c * 32, sr[c]);
        tmem_ld_wait();
        if ((warp & (4 * kH - 1)) == 0) FTRACE(tn, 4 * t + 2);
        const int col0 = j * FCP_TK + half * kCW;
        if (col0 + kCW - 1 > warp_min_limit) {      // diagonal / boundary tile: mask in registers
#pragma unroll
          for (int c = 0; c < kCW / 32; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (col0 + c * 32 + i > limit) sr[c][i] = 0xff800000u;   // -inf
        }
        // ---- fast path: exponentials against the running max, tile max on the side
        bool exact = (kH == 2) || j == 0 || __any_sync(0xffffffffu, m == -INFINITY);
        if (!exact) {
          float mx = -INFINITY, sum = 0.f;
#pragma unroll
          for (int c = 0; c < kCW / 32; ++c) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              uint32_t pk[8];
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const float s0 = __uint_as_float(sr[c][h * 16 + 2 * i]);
                const float s1 = __uint_as_float(sr[c][h * 16 + 2 * i + 1]);
                mx = fmaxf(mx, fmaxf(s0, s1));
                const float p0 = fast_exp2(fmaf(s0, scale_log2, -m));
                const float p1 = fast_exp2(fmaf(s1, scale_log2, -m));
                sum += p0 + p1;
                pk[i] = pack_bf16(p0, p1);
              }
              tmem_st8(tP + c * 16 + h * 8, pk);
            }
          }
          exact = __any_sync(0xffffffffu, mx * scale_log2 > m + kRescaleThreshold);
          if (!exact) l += sum;
        }
        if (exact) {
          // ---- exact path: tile max first (and over both halves when kH = 2)
          float mx = -INFINITY;
#pragma unroll
          for (int c = 0; c < kCW / 32; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(sr[c][i]));
          if (kH == 2) {
            // The barrier also orders this part's P stores (into columns the other part loaded
            // S from) after the other part's loads.
            *xch_mine = mx;
            named_bar_sync(pair_bar, 128 * kH);
            mx = fmaxf(mx, *xch_other);
          }
          const float m_new = fmaxf(m, mx * scale_log2);
          const bool grow = m_new > m + kRescaleThreshold;   // also first finite max (m = -inf)
          const bool any_grow = __any_sync(0xffffffffu, grow);
          float alpha = 1.f;
          if (grow) {
            alpha = fast_exp2(m - m_new);                   // m = -inf -> 0
            m = m_new;
          }
          const float m_use = (m == -INFINITY) ? 0.f : m;
          float sum = 0.f;
#pragma unroll
          for (int c = 0; c < kCW / 32; ++c) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              uint32_t pk[8];
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const float p0 = fast_exp2(fmaf(__uint_as_float(sr[c][h * 16 + 2 * i]), scale_log2, -m_use));
                const float p1 = fast_exp2(fmaf(__uint_as_float(sr[c][h * 16 + 2 * i + 1]), scale_log2, -m_use));
                sum += p0 + p1;
                pk[i] = pack_bf16(p0, p1);
              }
              tmem_st8(tP + c * 16 + h * 8, pk);
            }
          }
          l = l * alpha + sum;
          if (any_grow && j > 0) {                          // rescale this thread's columns of O
#pragma unroll
            for (int c = 0; c < kOW / 32; ++c) {
              uint32_t orow[32];
              tmem_ld32(tO + c * 32, orow);
              tmem_ld_wait();
#pragma unroll
              for (int i = 0; i < 32; ++i) orow[i] = __float_as_uint(__uint_as_float(orow[i]) * alpha);
              tmem_st32(tO + c * 32, orow);
            }
          }
        }
        tmem_st_wait();
        tc_fence_before();
        mbar_arrive(&bars->p_ready[t]);
        if ((warp & (4 * kH - 1)) == 0) FTRACE(tn, 4 * t + 3);
        if (warp == 5) FTRACE(tn, 14);
        if (warp == 7) FTRACE(tn, 15);
#ifdef FCP_EXP_TRACE
        ++tn;
#endif
      }

      // epilogue: o = O / l, lse = ln2 * (m + log2 l)
      if (kH == 2) {
        *xch_mine = l;
        named_bar_sync(pair_bar, 128 * kH);
        l += *xch_other;
      }
      mbar_wait(&bars->o_full[t], o_ph);
      o_ph ^= 1;
      tc_fence_after();
      const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
      for (int c = 0; c < kOW / 32; ++c) {
        uint32_t orow[32];
        tmem_ld32(tO + c * 32, orow);
        tmem_ld_wait();
        if (row_valid) {
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            int4 pk;
            pk.x = pack_bf16(__uint_as_float(orow[8 * i + 0]) * inv, __uint_as_float(orow[8 * i + 1]) * inv);
            pk.y = pack_bf16(__uint_as_float(orow[8 * i + 2]) * inv, __uint_as_float(orow[8 * i + 3]) * inv);
            pk.z = pack_bf16(__uint_as_float(orow[8 * i + 4]) * inv, __uint_as_float(orow[8 * i + 5]) * inv);
            pk.w = pack_bf16(__uint_as_float(orow[8 * i + 6]) * inv, __uint_as_float(orow[8 * i + 7]) * inv);
            *reinterpret_cast<int4*>(o_row + c * 32 + i * 8) = pk;
          }
        }
      }
      tc_fence_before();
      mbar_arrive(&bars->o_empty[t]);
      if (row_valid && half == 0) *lse_row = l > 0.f ? kLn2 * (m + __log2f(l)) : -INFINITY;
      // the exchange slot is rewritten at the next item's first tile: keep the parts together
      if (kH == 2) named_bar_sync(pair_bar, 128 * kH);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc<Cfg::kTmemCols>(tmem_base);
  }
}

template <int D, int NQ>
int launch_fwd(const fcp_attn_args* a, const fcp_sched* s) {
  using Cfg = FwdCfg<D, NQ>;
  CUtensorMap mq, mk, mv;
  if (!make_tmap_rows(&mq, a->q, D, s->Hq, s->n_q, 128) ||
      !make_tmap_rows(&mk, a->k, D, s->Hkv, s->n_kv, 128) ||
      !make_tmap_rows(&mv, a->v, D, s->Hkv, s->n_kv, 128))
    return FCP_CUDA;
  auto kern = fcp_attn_fwd_kernel<D, NQ>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes) !=
      cudaSuccess)
    return FCP_CUDA;
  const int grid = s->n_cta;
  const FwdItem* items =
      reinterpret_cast<const FwdItem*>(static_cast<const char*>(a->workspace) + s->off_fwd);
  cudaStream_t st = (cudaStream_t)a->stream;
  if (a->ev_start && cudaEventRecord((cudaEvent_t)a->ev_start, st) != cudaSuccess) return FCP_CUDA;
  kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, st>>>(
      mq, mk, mv, items,
      reinterpret_cast<const int32_t*>(static_cast<const char*>(a->workspace) + s->off_fwd_cta),
      static_cast<__nv_bfloat16*>(a->o), a->lse, s->n_q, s->Hq, a->scale * kLog2e);
  if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
  if (a->ev_stop && cudaEventRecord((cudaEvent_t)a->ev_stop, st) != cudaSuccess) return FCP_CUDA;
  return FCP_OK;
}

}  // namespace

extern "C" int fcp_attn_fwd(const fcp_attn_args* a) {
  if (!a || !a->sched || !a->workspace || !a->q || !a->k || !a->v || !a->o || !a->lse)
    return FCP_INVALID_ARG;
  const fcp_sched* s = a->sched;
  for (const void* p : {a->q, a->k, a->v, (const void*)a->o, (const void*)a->workspace})
    if (reinterpret_cast<uintptr_t>(p) & 15) return FCP_MISALIGNED;
  if (s->fwd.empty()) return FCP_OK;
  if (s->D == 128) return s->NQ == 2 ? launch_fwd<128, 2>(a, s) : launch_fwd<128, 1>(a, s);
  if (s->D == 64) return s->NQ == 2 ? launch_fwd<64, 2>(a, s) : launch_fwd<64, 1>(a, s);
  return FCP_UNSUPPORTED;
}
