// Document-masked causal attention forward for sm_100a.
//
// One persistent CTA per SM.  A work item is one 128-row q tile of one shard for a pack of NQ
// query heads that share a kv head (GQA): the NQ tiles share every K/V tile staged in shared
// memory and ping-pong on the tensor core — while the softmax warpgroup of one tile works, the
// MMAs of the other tile run.
//
//   warp 0      TMA producer   Q (once per item), K/V tiles through a ring of smem stages
//   warp 1      MMA issuer     S_t = Q_t K^T (SS), O_t += P_t V (A = P from TMEM, B = V MN-major)
//   warps 4..   softmax        one warpgroup per q tile, one query row per thread: mask from
//                              (q_pos0 + row, kv_len), online softmax with lazy rescale of O,
//                              P written back to TMEM as bf16 over S, epilogue o = O / l
//
// TMEM columns: S_t at 128 t, O_t at 128 (NQ + t); P_t aliases the first 64 columns of S_t.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "fcp_internal.h"
#include "fcp_sm100.cuh"
#include "fcp_tma.h"

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
  static constexpr int kThreads = 128 + 128 * NQ;
  static constexpr int kTmemCols = 256 * NQ;
  static constexpr int kSmemData = (NQ + kStages) * kTileBytes;
  static constexpr int kSmemBytes = 1024 + kSmemData + 1024;
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
  FwdBarriers* bars = reinterpret_cast<FwdBarriers*>(smem + Cfg::kSmemData);

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
      mbar_init(&bars->p_ready[t], 128);
      mbar_init(&bars->o_full[t], 1);
      mbar_init(&bars->o_empty[t], 128);
    }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<Cfg::kTmemCols>(&bars->tmem_base);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;
  const int item_begin = cta_off[blockIdx.x], item_end = cta_off[blockIdx.x + 1];   // this CTA's work list

  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    if (lane == 0) {
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
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ MMA issuer
    // The whole warp walks the loop and waits on the barriers; one elected lane issues the
    // tcgen05 instructions (a converged warp + elect.sync compiles to straight-line UTCHMMA).
    constexpr uint32_t idesc_qk = umma_idesc_bf16(128, 128, 0, 0);
    constexpr uint32_t idesc_pv = umma_idesc_bf16(128, D, 0, 1);
    const uint64_t q_desc0 = umma_desc_sw128(smem_u32(q_smem), 16, 1024);          // K-major
    const uint64_t ring_kmaj = umma_desc_sw128(smem_u32(ring), 16, 1024);          // K tile
    const uint64_t ring_mnmaj = umma_desc_sw128(smem_u32(ring), Cfg::kPanelBytes, 1024);  // V tile
    uint32_t kv_n = 0, item_n = 0, p_ph[2] = {0, 0};

    auto issue_qk = [&](int t, uint32_t kslot) {
      const uint64_t a0 = umma_desc_add(q_desc0, t * Cfg::kTileBytes);
      const uint64_t b0 = umma_desc_add(ring_kmaj, kslot * Cfg::kTileBytes);
#pragma unroll
      for (int kk = 0; kk < D / 16; ++kk) {
        const uint32_t off = (kk >> 2) * Cfg::kPanelBytes + (kk & 3) * 32;
        umma_ss(tmem_base + t * 128, umma_desc_add(a0, off), umma_desc_add(b0, off), idesc_qk,
                kk > 0);
      }
    };
    auto issue_pv = [&](int t, uint32_t vslot, bool acc) {
      const uint64_t b0 = umma_desc_add(ring_mnmaj, vslot * Cfg::kTileBytes);
#pragma unroll
      for (int kk = 0; kk < 128 / 16; ++kk)
        umma_ts(tmem_base + (NQ + t) * 128, tmem_base + t * 128 + kk * 8,
                umma_desc_add(b0, kk * 2048), idesc_pv, (acc || kk > 0) ? 1u : 0u);
    };

    for (int idx = item_begin; idx < item_end; ++idx) {
      const FwdItem it = items[idx];
      const int n = it.n_kv_tiles;
      if (n == 0) continue;
      mbar_wait(&bars->q_full, item_n & 1);
      {
        const uint32_t kslot = kv_n % Cfg::kStages;
        mbar_wait(&bars->kv_full[kslot], (kv_n / Cfg::kStages) & 1);
        tc_fence_after();
        if (elect_one()) {
          for (int t = 0; t < NQ; ++t) {
            issue_qk(t, kslot);
            umma_commit(&bars->s_full[t]);
          }
          umma_commit(&bars->kv_empty[kslot]);
          if (n == 1) umma_commit(&bars->q_empty);
        }
        __syncwarp();
        ++kv_n;
      }
      for (int j = 0; j < n; ++j) {
        const bool has_next = j + 1 < n;
        const uint32_t vslot = kv_n % Cfg::kStages, vph = (kv_n / Cfg::kStages) & 1;
        const uint32_t kslot = (kv_n + 1) % Cfg::kStages,
                       kph = ((kv_n + 1) / Cfg::kStages) & 1;
        for (int t = 0; t < NQ; ++t) {
          mbar_wait(&bars->p_ready[t], p_ph[t]);
          p_ph[t] ^= 1;
          if (j == 0) mbar_wait(&bars->o_empty[t], (item_n & 1) ^ 1);
          if (t == 0) {
            mbar_wait(&bars->kv_full[vslot], vph);
            if (has_next) mbar_wait(&bars->kv_full[kslot], kph);
          }
          tc_fence_after();
          if (elect_one()) {
            issue_pv(t, vslot, j > 0);
            if (has_next) {
              issue_qk(t, kslot);
              umma_commit(&bars->s_full[t]);
            } else {
              umma_commit(&bars->o_full[t]);
            }
          }
          __syncwarp();
        }
        if (elect_one()) {
          umma_commit(&bars->kv_empty[vslot]);
          if (has_next) {
            umma_commit(&bars->kv_empty[kslot]);
            if (j + 2 == n) umma_commit(&bars->q_empty);
          }
        }
        __syncwarp();
        kv_n += has_next ? 2 : 1;
      }
      ++item_n;
    }
  } else if (warp >= 4) {
    // ------------------------------------------------------------------ softmax + epilogue
    const int t = (warp - 4) >> 2;                 // q tile of this warpgroup
    const int row = (warp & 3) * 32 + lane;        // query row = TMEM lane
    const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem_base + lane_addr + t * 128;
    const uint32_t tO = tmem_base + lane_addr + (NQ + t) * 128;
    uint32_t s_ph = 0, o_ph = 0;

    for (int idx = item_begin; idx < item_end; ++idx) {
      const FwdItem it = items[idx];
      const int n = it.n_kv_tiles;
      const int head = it.head0 + t;
      const bool row_valid = row < it.q_rows;
      __nv_bfloat16* o_row = o + ((int64_t)(it.q_row0 + row) * Hq + head) * D;
      float* lse_row = lse + (int64_t)head * n_q + it.q_row0 + row;
      if (n == 0) {                                 // no visible key: o = 0, lse = -inf
        if (row_valid) {
          for (int c = 0; c < D; c += 8) *reinterpret_cast<int4*>(o_row + c) = make_int4(0, 0, 0, 0);
          *lse_row = -INFINITY;
        }
        continue;
      }
      // last visible key (segment position) of this row; may be negative
      const int limit = min(it.q_pos0 + row, it.kv_len - 1);
      const int warp_min_limit = min(it.q_pos0 + (warp & 3) * 32, it.kv_len - 1);
      float m = -INFINITY, l = 0.f;

      for (int j = 0; j < n; ++j) {
        mbar_wait(&bars->s_full[t], s_ph);
        s_ph ^= 1;
        tc_fence_after();
        uint32_t sr[4][32];
#pragma unroll
        for (int c = 0; c < 4; ++c) tmem_ld32(tS + c * 32, sr[c]);
        tmem_ld_wait();
        const int col0 = j * FCP_TK;
        if (col0 + FCP_TK - 1 > warp_min_limit) {   // diagonal / boundary tile: mask in registers
#pragma unroll
          for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (col0 + c * 32 + i > limit) sr[c][i] = 0xff800000u;   // -inf
        }
        float mx = -INFINITY;
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
          for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(sr[c][i]));
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
        for (int c = 0; c < 4; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const float p0 = fast_exp2(fmaf(__uint_as_float(sr[c][2 * i]), scale_log2, -m_use));
            const float p1 = fast_exp2(fmaf(__uint_as_float(sr[c][2 * i + 1]), scale_log2, -m_use));
            sum += p0 + p1;
            pk[i] = pack_bf16(p0, p1);
          }
          tmem_st16(tS + c * 16, pk);
        }
        l = l * alpha + sum;
        if (any_grow && j > 0) {                          // rescale the running O row
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t orow[32];
            tmem_ld32(tO + c * 32, orow);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) orow[i] = __float_as_uint(__uint_as_float(orow[i]) * alpha);
            tmem_st32(tO + c * 32, orow);
          }
        }
        tmem_st_wait();
        tc_fence_before();
        mbar_arrive(&bars->p_ready[t]);
      }

      // epilogue: o = O / l, lse = ln2 * (m + log2 l)
      mbar_wait(&bars->o_full[t], o_ph);
      o_ph ^= 1;
      tc_fence_after();
      const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
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
      if (row_valid) *lse_row = l > 0.f ? kLn2 * (m + __log2f(l)) : -INFINITY;
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
