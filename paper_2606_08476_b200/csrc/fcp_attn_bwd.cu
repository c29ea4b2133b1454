// Document-masked causal attention backward (formulas in include/fcp.h)
// for sm_100a.
//
// Three launches:
//   1. fcp_bwd_prep      zeroes the fp32 dq accumulator; delta = rowsum(dO o O); (lse*log2e, delta) into a 64-row-padded scratch
//                        so that every q tile's statistics are one aligned 512-byte bulk copy;
//                        padding rows get lse = +inf (P = 0: they contribute nothing).
//   2. fcp_attn_bwd_main one persistent CTA per SM, 16 warps.  A work item is one 128-row KV
//                        tile of one KV segment for one kv head; it loops over every (shard,
//                        64-row q tile, query head of the GQA group) that sees the tile and keeps
//                        dK, dV in TMEM for the whole item (the GQA sum costs nothing, no atomics):
//      (roles; the control warpgroup is mapped to the highest warp ids, see the kernel)
//        role 0      TMA producer  K,V tile once per item; Q, dO, (lse,delta) per iteration (3 stages)
//        role 1      MMA issuer    S^T = K Q^T, dP^T = V dO^T (SS);  dV += P^T dO, dK += dS^T Q
//                                  (A from TMEM);  dQ^T = K^T dS^T (SS, dS^T staged in smem)
//        warps 4-11  softmax       two warpgroups, 32 q columns each, one KV row per thread:
//                                  P^T = exp2(S^T c - lse), mask, dS^T = P^T o (dP^T - delta);
//                                  bf16 P^T/dS^T back into TMEM, dS^T also into swizzled smem
//        warps 12-15 dQ drain      TMEM -> smem (transposed) -> cp.reduce.async.bulk add.f32
//                                  into the fp32 dq accumulator [Hq][padded rows][D]
//   3. fcp_bwd_dq_convert dq = bf16(scale * accumulator)
//
// TMEM columns: S^T[2] at 0/64 (after softmax, per 32-column half: P^T in its first 16 columns,
// dS^T in its last 16),
// dP^T at 128, dQ^T at 192, dV at 256, dK at 384.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <atomic>

#include "fcp_internal.h"
#include "fcp_sm100.cuh"
#include "fcp_tma.h"

namespace {
using namespace fcp;

constexpr float kLog2e = 1.4426950408889634f;

// ------------------------------------------------------------------------------------------
// 1. prepass
// ------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256)
fcp_bwd_prep(const __nv_bfloat16* __restrict__ o, const __nv_bfloat16* __restrict__ dO,
             const float* __restrict__ lse, const int32_t* __restrict__ tile_meta,
             float2* __restrict__ lsed, float4* __restrict__ dq_acc, int64_t n_q, int64_t n_q_pad,
             int Hq) {
  const int tile = blockIdx.x, head = blockIdx.y;
  // zero this (q tile, head) block of the fp32 dQ accumulator: saves a separate memset pass
  // (dq_acc == nullptr: the accumulator holds an earlier KV piece's partial, FCP_DQ_KEEP)
  if (dq_acc != nullptr) {
    float4* z = dq_acc + ((int64_t)head * n_q_pad + (int64_t)tile * FCP_BQ) * (D / 4);
    for (int i = threadIdx.x; i < FCP_BQ * D / 4; i += blockDim.x) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  const int row0 = tile_meta[2 * tile], valid = tile_meta[2 * tile + 1];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  constexpr int kPerLane = D / 32;                       // 2 or 4 bf16 per lane
  for (int r = warp; r < FCP_BQ; r += 8) {
    float2 out = make_float2(INFINITY, 0.f);
    if (r < valid) {
      const int64_t base = ((int64_t)(row0 + r) * Hq + head) * D + lane * kPerLane;
      float acc = 0.f;
#pragma unroll
      for (int i = 0; i < kPerLane; i += 2) {
        const float2 a = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(o + base + i));
        const float2 b = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(dO + base + i));
        acc += a.x * b.x + a.y * b.y;
      }
#pragma unroll
      for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
      const float l = lse[(int64_t)head * n_q + row0 + r];
      out = make_float2(l == -INFINITY ? INFINITY : l * kLog2e, acc);
    }
    if (lane == 0) lsed[(int64_t)head * n_q_pad + (int64_t)tile * FCP_BQ + r] = out;
  }
}

// ------------------------------------------------------------------------------------------
// 3. dq convert
// ------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256)
fcp_bwd_dq_convert(const float* __restrict__ acc, const int32_t* __restrict__ tile_meta,
                   __nv_bfloat16* __restrict__ dq, int64_t n_q_pad, int Hq, float scale) {
  const int tile = blockIdx.x, head = blockIdx.y;
  const int row0 = tile_meta[2 * tile], valid = tile_meta[2 * tile + 1];
  constexpr int kVecPerRow = D / 8;
  for (int idx = threadIdx.x; idx < valid * kVecPerRow; idx += blockDim.x) {
    const int r = idx / kVecPerRow, c = (idx % kVecPerRow) * 8;
    const float* src = acc + ((int64_t)head * n_q_pad + (int64_t)tile * FCP_BQ + r) * D + c;
    const float4 a = *reinterpret_cast<const float4*>(src);
    const float4 b = *reinterpret_cast<const float4*>(src + 4);
    int4 pk;
    pk.x = pack_bf16(a.x * scale, a.y * scale);
    pk.y = pack_bf16(a.z * scale, a.w * scale);
    pk.z = pack_bf16(b.x * scale, b.y * scale);
    pk.w = pack_bf16(b.z * scale, b.w * scale);
    *reinterpret_cast<int4*>(dq + ((int64_t)(row0 + r) * Hq + head) * D + c) = pk;
  }
}

// ------------------------------------------------------------------------------------------
// 2. main kernel
// ------------------------------------------------------------------------------------------
template <int D>
struct BwdCfg {
  static constexpr int kPanels = D / 64;
  static constexpr int kKVTile = 128 * D * 2;            // K or V tile: kPanels x [128 rows x 128 B]
  static constexpr int kKVPanel = 128 * 128;
  static constexpr int kQTile = FCP_BQ * D * 2;          // Q or dO tile: kPanels x [64 rows x 128 B]
  static constexpr int kQPanel = FCP_BQ * 128;
  static constexpr int kStat = FCP_BQ * 8;               // (lse, delta) of one q tile
  static constexpr int kStage = 2 * kQTile;              // Q, dO
  static constexpr int kStages = 3;
  static constexpr int kDS = 128 * 128;                  // dS^T bf16 [128 kv][64 q]
  static constexpr int kDQ = FCP_BQ * D * 4;             // dQ staging fp32 [64 q][D]
  static constexpr int kThreads = 512;                   // 4 warpgroups: control, softmax x2, dQ drain
  static constexpr int kOffKV = 0;
  static constexpr int kOffStage = 2 * kKVTile;
  static constexpr int kOffDS = kOffStage + kStages * kStage;
  static constexpr int kOffDQ = kOffDS + 2 * kDS;
  static constexpr int kOffStat = kOffDQ + kDQ;
  static constexpr int kOffBar = kOffStat + kStages * kStat;
  static constexpr int kSmemBytes = 1024 + kOffBar + 256;
  static constexpr uint32_t kStageTx = 2 * kQTile + kStat;
  // TMEM columns
  static constexpr int kColS = 0, kColDP = 128, kColDQ = 192, kColDV = 256, kColDK = 384;
  // registers per thread after setmaxnreg (launch: 128): control, softmax x2, drain
  static constexpr int kRegsCtl = 96, kRegsSoftmax = 152, kRegsDrain = 104;
};
static_assert(BwdCfg<128>::kSmemBytes <= 232448, "bwd shared memory exceeds 227 KB");

struct BwdBarriers {
  uint64_t kv_full, kv_free;
  uint64_t qdo_full[3], qdo_free[3];
  uint64_t st_full, p_ready;
  uint64_t ds_free[2];
  uint64_t dq_full, dq_free;
  uint64_t dkv_full, dkv_free;
  uint32_t tmem_base;
};
static_assert(sizeof(BwdBarriers) <= 256, "barrier block");

// Enumerates the inner iterations of an item in the one order every warp role follows:
// shards seen by the KV tile -> 64-row q tiles -> the G query heads of the kv head.
struct IterWalk {
  const BwdSub* subs;
  int sub, sub_end, qt, n_qt, g, G;
  BwdSub cur;
  __device__ IterWalk(const BwdItem& it, const BwdSub* all, int G_)
      : subs(all), sub(it.sub_begin), sub_end(it.sub_end), qt(0), n_qt(0), g(0), G(G_) {
    if (sub < sub_end) {
      cur = subs[sub];
      n_qt = (cur.q_rows + FCP_BQ - 1) / FCP_BQ;
    }
  }
  __device__ bool done() const { return sub >= sub_end; }
  __device__ int q_row() const { return cur.q_row0 + qt * FCP_BQ; }
  __device__ int q_pos() const { return cur.q_pos0 + qt * FCP_BQ; }
  __device__ int pad_row() const { return cur.pad_row0 + qt * FCP_BQ; }
  __device__ int valid() const { return min(FCP_BQ, cur.q_rows - qt * FCP_BQ); }
  __device__ void next() {
    if (++g < G) return;
    g = 0;
    if (++qt < n_qt) return;
    qt = 0;
    if (++sub < sub_end) {
      cur = subs[sub];
      n_qt = (cur.q_rows + FCP_BQ - 1) / FCP_BQ;
    }
  }
};

__device__ __forceinline__ void bulk_reduce_add_f32(float* gdst, const void* ssrc, uint32_t bytes) {
  asm volatile(
      "cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(gdst),
      "r"(smem_u32(ssrc)), "r"(bytes)
      : "memory");
}
// 3-D tiled store shared -> global through a tensor map (coordinates as tma_load_3d)
__device__ __forceinline__ void tma_store_3d(const void* tmap, uint32_t smem_src, int32_t c0,
                                             int32_t c1, int32_t c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::
                   "l"(tmap), "r"(smem_src), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() {
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read0() {
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait0() {
  asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// One softmax step of the backward for one KV row (= one thread) and 32 query columns
// (the two softmax warpgroups take the two halves of a 64-column q tile):
//   P^T = exp2(S^T c - lse), masked;  dS^T = P^T o (dP^T - delta)
// bf16 P^T / dS^T go back into TMEM (A operands of dV / dK) and dS^T into the swizzled smem tile
// (B operand of dQ^T).  kMask selects the diagonal / ragged-tile variant; interior tiles skip
// every mask instruction.
template <bool kMask>
__device__ __forceinline__ void bwd_softmax_half(const uint32_t (&s)[32], const uint32_t (&dp)[32],
                                                 uint32_t stat_addr, float scale_log2,
                                                 int vis,   // kMask: columns c < vis are masked out
                                                 uint32_t tP, uint32_t tDS, uint32_t ds_row_addr,
                                                 int chunk0, int row) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {                       // 16 columns per step
    uint32_t pk_p[8], pk_ds[8];
#pragma unroll
    for (int i = 0; i < 16; i += 2) {
      const int c = h * 16 + i;
      const float4 st01 = lds128(stat_addr + c * 8);  // lse0, delta0, lse1, delta1
      float p0 = fast_exp2(fmaf(__uint_as_float(s[c]), scale_log2, -st01.x));
      float p1 = fast_exp2(fmaf(__uint_as_float(s[c + 1]), scale_log2, -st01.z));
      if (kMask) {
        if (c < vis) p0 = 0.f;
        if (c + 1 < vis) p1 = 0.f;
      }
      const float ds0 = p0 * (__uint_as_float(dp[c]) - st01.y);
      const float ds1 = p1 * (__uint_as_float(dp[c + 1]) - st01.w);
      pk_p[i >> 1] = pack_bf16(p0, p1);
      pk_ds[i >> 1] = pack_bf16(ds0, ds1);
    }
    tmem_st8(tP + h * 8, pk_p);
    tmem_st8(tDS + h * 8, pk_ds);
#pragma unroll
    for (int c4 = 0; c4 < 2; ++c4) {                  // two 16-byte chunks of the 128-byte row
      const int chunk = (chunk0 + h * 2 + c4) ^ (row & 7);
      sts128(ds_row_addr + chunk * 16, pk_ds[4 * c4], pk_ds[4 * c4 + 1], pk_ds[4 * c4 + 2],
             pk_ds[4 * c4 + 3]);
    }
  }
}

template <int D>
__global__ void __launch_bounds__(BwdCfg<D>::kThreads, 1)
fcp_attn_bwd_main(const __grid_constant__ CUtensorMap tmap_q,
                  const __grid_constant__ CUtensorMap tmap_do,
                  const __grid_constant__ CUtensorMap tmap_k,
                  const __grid_constant__ CUtensorMap tmap_v,
                  const __grid_constant__ CUtensorMap tmap_dk,
                  const __grid_constant__ CUtensorMap tmap_dv,
                  const BwdItem* __restrict__ items, const int32_t* __restrict__ cta_off,
                  const BwdSub* __restrict__ subs, const float2* __restrict__ lsed,
                  float* __restrict__ dq_acc, void* __restrict__ dk_out,
                  void* __restrict__ dv_out, int dkv_f32, int64_t n_q_pad, int Hkv, int G,
                  float scale, float scale_log2) {
  using Cfg = BwdCfg<D>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) &
                                             ~uintptr_t(1023));
  uint8_t* k_smem = smem + Cfg::kOffKV;
  uint8_t* v_smem = k_smem + Cfg::kKVTile;
  uint8_t* stage_smem = smem + Cfg::kOffStage;
  uint8_t* ds_smem = smem + Cfg::kOffDS;
  uint8_t* dq_smem = smem + Cfg::kOffDQ;
  uint8_t* stat_smem = smem + Cfg::kOffStat;
  BwdBarriers* bars = reinterpret_cast<BwdBarriers*>(smem + Cfg::kOffBar);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  // Role of the warp.  The control warpgroup sits in the HIGHEST warp ids (12-15): the warp
  // scheduler favours high ids, and the single MMA-issuing thread must never queue behind the
  // softmax warps of its sub-partition.  TMEM lane quarters depend on warp % 4 only.
  const int role = (warp + 4) & 15;   // 0 producer, 1 MMA, 4-11 softmax, 12-15 dQ drain

  if (threadIdx.x == 0) {
    mbar_init(&bars->kv_full, 1);
    mbar_init(&bars->kv_free, 1);
    for (int i = 0; i < Cfg::kStages; ++i) {
      // the producer's arrive.expect_tx plus the 256 softmax threads: stage i is "full" for the
      // MMA thread when Q, dO and the statistics have landed AND the previous iteration's S^T /
      // dP^T sit in registers (dP^T has one TMEM buffer): ONE wait gates [S^T, dP^T](n+1)
      mbar_init(&bars->qdo_full[i], 257);
      mbar_init(&bars->qdo_free[i], 1);
    }
    for (int i = 0; i < 2; ++i) mbar_init(&bars->ds_free[i], 1);
    mbar_init(&bars->st_full, 1);
    mbar_init(&bars->p_ready, 256);
    mbar_init(&bars->dq_full, 1);
    mbar_init(&bars->dq_free, 128);
    mbar_init(&bars->dkv_full, 1);
    mbar_init(&bars->dkv_free, 256);
    fence_barrier_init();
  }
  if (role == 1) tmem_alloc<512>(&bars->tmem_base);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;
  const int item_begin = cta_off[blockIdx.x], item_end = cta_off[blockIdx.x + 1];   // this CTA's work list

  if (role < 4) {
    reg_dealloc<Cfg::kRegsCtl>();
    if (role == 0 && lane == 0) {
      // ---------------------------------------------------------------- TMA producer
      prefetch_tmap(&tmap_q);
      prefetch_tmap(&tmap_do);
      prefetch_tmap(&tmap_k);
      prefetch_tmap(&tmap_v);
      uint32_t n = 0, m = 0;          // global iteration / item counters
      for (int idx = item_begin; idx < item_end; ++idx) {
        const BwdItem it = items[idx];
        if (it.n_iters == 0) continue;
        mbar_wait(&bars->kv_free, (m & 1) ^ 1);
        mbar_arrive_expect_tx(&bars->kv_full, 2 * Cfg::kKVTile);
        for (int pn = 0; pn < Cfg::kPanels; ++pn) {
          tma_load_3d(k_smem + pn * Cfg::kKVPanel, &tmap_k, &bars->kv_full, pn * 64, it.kv_head,
                      it.kv_row0);
          tma_load_3d(v_smem + pn * Cfg::kKVPanel, &tmap_v, &bars->kv_full, pn * 64, it.kv_head,
                      it.kv_row0);
        }
        for (IterWalk w(it, subs, G); !w.done(); w.next(), ++n) {
          const uint32_t st = n % Cfg::kStages;
          uint8_t* sq = stage_smem + st * Cfg::kStage;
          const int head = it.kv_head * G + w.g;
          mbar_wait(&bars->qdo_free[st], ((n / Cfg::kStages) & 1) ^ 1);
          mbar_arrive_expect_tx(&bars->qdo_full[st], Cfg::kStageTx);
          for (int pn = 0; pn < Cfg::kPanels; ++pn) {
            tma_load_3d(sq + pn * Cfg::kQPanel, &tmap_q, &bars->qdo_full[st], pn * 64, head,
                        w.q_row());
            tma_load_3d(sq + Cfg::kQTile + pn * Cfg::kQPanel, &tmap_do, &bars->qdo_full[st],
                        pn * 64, head, w.q_row());
          }
          bulk_load_1d(stat_smem + st * Cfg::kStat, lsed + (int64_t)head * n_q_pad + w.pad_row(),
                       Cfg::kStat, &bars->qdo_full[st]);
        }
        ++m;
      }
    } else if (role == 1 && elect_one()) {
      // ---------------------------------------------------------------- MMA issuer
      // One elected thread (elect.sync compiles to straight-line UTCHMMA).  The tcgen05 queue is
      // only about 5 MMAs deep, so issue runs at the pace of execution and every barrier the
      // thread looks at costs the pipe 90-150 clocks once the queue has drained: it looks at
      // THREE per iteration (stage full + dP^T free in one, p_ready, dq_free right before the
      // dQ^T product) with plain try_wait loops.  Round 1 probed five with mbarrier.test_wait
      // ahead of time; a trace showed the probes themselves (~150 clocks each) were the larger
      // cost: 8b 1000 -> 1038 TFLOP/s.  All per-iteration scalar work is a handful of 32-bit
      // adds on precomputed descriptor words.
      constexpr uint32_t idesc_s = umma_idesc_bf16(128, FCP_BQ, 0, 0);    // S^T, dP^T
      constexpr uint32_t idesc_kv = umma_idesc_bf16(128, D, 0, 1);        // dV, dK
      constexpr uint32_t idesc_dq = umma_idesc_bf16(128, FCP_BQ, 1, 1);   // dQ^T
      constexpr int kSteps = D / 16;
      // Every operand here uses SWIZZLE_128B with SBO = 1024: the high descriptor word is one
      // constant, the low word is (address >> 4) | (LBO >> 4) << 16.
      constexpr uint32_t kHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO, version, swizzle
      auto lo_word = [](uint32_t saddr, uint32_t lbo) { return ((saddr & 0x3FFFF) >> 4) | ((lbo >> 4) << 16); };
      auto desc = [](uint32_t lo) { return ((uint64_t)kHi << 32) | lo; };
      const uint32_t k_kmaj = lo_word(smem_u32(k_smem), 16);                 // A of S^T
      const uint32_t v_kmaj = lo_word(smem_u32(v_smem), 16);                 // A of dP^T
      const uint32_t k_mnmaj = lo_word(smem_u32(k_smem), Cfg::kKVPanel);     // A of dQ^T
      const uint32_t ds_mnmaj = lo_word(smem_u32(ds_smem), 1024);            // B of dQ^T (buffer 0)
      const uint32_t q_kmaj0 = lo_word(smem_u32(stage_smem), 16);            // B of S^T  (stage 0)
      const uint32_t q_mnmaj0 = lo_word(smem_u32(stage_smem), Cfg::kQPanel); // B of dK   (stage 0)
      constexpr uint32_t kStageStep = Cfg::kStage >> 4, kDoStep = Cfg::kQTile >> 4;
      // ring state of iteration n: stage index, parity of the stage's phase, n & 1
      uint32_t st = 0, sph = 0, b = 0, mph = 0;

      // Keeps ptxas from hoisting the eight 64-bit A descriptors of a product out of the loop
      // into general registers (16 R2UR per product and iteration); from an opaque base they
      // are one R2UR plus uniform adds, like the B descriptors.
      auto opaque = [](uint32_t x) {
        asm volatile("" : "+r"(x));
        return x;
      };
      // S^T = K Q^T  or  dP^T = V dO^T : A = kv tile (K-major), B = q/dO tile (K-major)
      auto issue_kq = [&](uint32_t d_col, uint32_t a_lo, uint32_t b_lo, int kk0, int kk1) {
#pragma unroll
        for (int kk = kk0; kk < kk1; ++kk)
          umma_ss(tmem_base + d_col,
                  desc(a_lo + (((kk >> 2) * Cfg::kKVPanel + (kk & 3) * 32) >> 4)),
                  desc(b_lo + (((kk >> 2) * Cfg::kQPanel + (kk & 3) * 32) >> 4)), idesc_s, kk > 0);
      };

      for (int idx = item_begin; idx < item_end; ++idx) {
        const int I = items[idx].n_iters;
        if (I == 0) continue;
        mbar_wait(&bars->kv_full, mph);
        // prologue: S^T and dP^T of the item's first iteration
        {
          mbar_wait(&bars->qdo_full[st], sph);
          tc_fence_after();
          const uint32_t q_lo = q_kmaj0 + st * kStageStep;
          issue_kq(Cfg::kColS + b * 64, k_kmaj, q_lo, 0, kSteps);
          issue_kq(Cfg::kColDP, v_kmaj, q_lo + kDoStep, 0, kSteps);
          umma_commit(&bars->st_full);
        }
        for (int i = 0; i < I; ++i) {
          // ring state of iterations n+1 and n+2
          const uint32_t st1 = st + 1 == Cfg::kStages ? 0 : st + 1, sph1 = st + 1 == Cfg::kStages ? sph ^ 1 : sph;
          if (i + 1 < I) {                       // next iteration's S^T / dP^T run ahead
            mbar_wait(&bars->qdo_full[st1], sph1);   // operands landed, dP^T(n) in registers
            tc_fence_after();
            const uint32_t q_lo = q_kmaj0 + st1 * kStageStep;
            const uint32_t v_lo = opaque(v_kmaj);
            issue_kq(Cfg::kColS + (b ^ 1) * 64, opaque(k_kmaj), q_lo, 0, kSteps);
            issue_kq(Cfg::kColDP, v_lo, q_lo + kDoStep, 0, kSteps);
            umma_commit(&bars->st_full);
          }
          mbar_wait(&bars->p_ready, b);
          if (i == 0) mbar_wait(&bars->dkv_free, mph ^ 1);
          tc_fence_after();
          // P^T / dS^T of q columns [32h, 32h+32) live in columns [32h, 32h+16) / [32h+16, 32h+32)
          // of the S^T buffer: each softmax warpgroup overwrites only the columns it has loaded
          const uint32_t tP = tmem_base + Cfg::kColS + b * 64, tDS = tP + 16;
          // dV += P^T dO, dK += dS^T Q : A from TMEM, B = dO / Q tile as MN-major [K=q][N=D]
          const uint32_t q_lo = q_mnmaj0 + st * kStageStep, do_lo = q_lo + kDoStep;
#pragma unroll
          for (int kk = 0; kk < FCP_BQ / 16; ++kk)
            umma_ts(tmem_base + Cfg::kColDV, tP + (kk >> 1) * 32 + (kk & 1) * 8,
                    desc(do_lo + kk * (2048 >> 4)), idesc_kv, (i > 0 || kk > 0) ? 1u : 0u);
#pragma unroll
          for (int kk = 0; kk < FCP_BQ / 16; ++kk)
            umma_ts(tmem_base + Cfg::kColDK, tDS + (kk >> 1) * 32 + (kk & 1) * 8,
                    desc(q_lo + kk * (2048 >> 4)), idesc_kv, (i > 0 || kk > 0) ? 1u : 0u);
          // dQ^T = K^T dS^T : A = K tile as MN-major [K=kv][M=d], B = dS^T smem MN-major [K=kv][N=q]
          const uint32_t ds_lo = ds_mnmaj + b * (Cfg::kDS >> 4);
          const uint32_t kt_lo = opaque(k_mnmaj);
          mbar_wait(&bars->dq_free, b ^ 1);          // the drain holds dQ^T(n-1) in registers
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)
            umma_ss(tmem_base + Cfg::kColDQ, desc(kt_lo + kk * (2048 >> 4)),
                    desc(ds_lo + kk * (2048 >> 4)), idesc_dq, kk > 0);
          umma_commit(&bars->qdo_free[st]);
          umma_commit(&bars->ds_free[b]);
          umma_commit(&bars->dq_full);
          st = st1;
          sph = sph1;
          b ^= 1;
        }
        umma_commit(&bars->dkv_full);
        umma_commit(&bars->kv_free);
        mph ^= 1;
      }
    }
  } else if (role < 12) {
    // ------------------------------------------------------------------ softmax / dS
    // Two warpgroups: warps 4-7 take q columns 0..31 of the 64-column tile, warps 8-11 take
    // columns 32..63 (a warp reaches TMEM lanes 32*(warp%4)..+31 only, so each warpgroup covers
    // all 128 KV rows).
    reg_alloc<Cfg::kRegsSoftmax>();
    mbar_arrive(&bars->qdo_full[0]);                   // dP^T is free before the first iteration
    const int half = (role - 4) >> 2;                  // 0 or 1
    const int row = (warp & 3) * 32 + lane;            // KV row of the tile = TMEM lane
    const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t stat_base = smem_u32(stat_smem) + half * 32 * 8;
    const uint32_t ds_base = smem_u32(ds_smem) + row * 128;
    const bool issuer = (warp & 3) == 0 && lane == 0;  // one thread per warpgroup issues its TMA stores
    bool staged = false;
    uint32_t n = 0, m = 0;
    for (int idx = item_begin; idx < item_end; ++idx) {
      const BwdItem it = items[idx];
      const bool row_valid = row < it.kv_rows;
      // output row of this thread (half 0 writes dv, half 1 writes dk), bf16 or fp32 elements
      const int64_t row_elem = ((int64_t)(it.kv_row0 + row) * Hkv + it.kv_head) * D;
      const int esz = dkv_f32 ? 4 : 2;
      uint8_t* dst_b = static_cast<uint8_t*>(half == 0 ? dv_out : dk_out) + row_elem * esz;
      if (it.n_iters == 0) {                             // no query sees this tile
        if (row_valid)
          for (int c = 0; c < D * esz; c += 16) *reinterpret_cast<int4*>(dst_b + c) = make_int4(0, 0, 0, 0);
        continue;
      }
      const int kv_pos = it.kv_pos0 + row;
      const int warp_kv_max = it.kv_pos0 + (warp & 3) * 32 + 31;
      if (staged) {
        // the previous item's dk / dv left through the dS^T buffers: both stores must have read
        // them before any softmax thread writes dS^T again
        if (issuer) bulk_wait_read0();
        named_bar_sync(6, 256);
        staged = false;
      }
      for (IterWalk w(it, subs, G); !w.done(); w.next(), ++n) {
        const uint32_t st = n % Cfg::kStages;
        const uint32_t tS = tmem_base + lane_addr + Cfg::kColS + (n & 1) * 64;
        const uint32_t tDP = tmem_base + lane_addr + Cfg::kColDP;
        const int q_pos = w.q_pos() + half * 32;       // position of this half's first column
        // mask needed when some (kv, q) pair of this warp's rows is invisible
        const bool need_mask = (warp_kv_max > q_pos) || (it.kv_rows < 128);
        mbar_wait(&bars->st_full, n & 1);
        tc_fence_after();
        uint32_t s[32], dp[32];
        tmem_ld32(tS + half * 32, s);
        tmem_ld32(tDP + half * 32, dp);
        mbar_wait(&bars->qdo_full[st], (n / Cfg::kStages) & 1);   // (lse, delta) of the q tile landed
        mbar_wait(&bars->ds_free[n & 1], ((n >> 1) & 1) ^ 1);     // dQ^T(n-2) has read dS^T smem
        tmem_ld_wait();
        tc_fence_before();
        // dP^T (and S^T) now in registers: counts towards the next iteration's stage barrier
        mbar_arrive(&bars->qdo_full[(n + 1) % Cfg::kStages]);
        const uint32_t stat_addr = stat_base + st * Cfg::kStat;
        const uint32_t ds_row_addr = ds_base + (n & 1) * Cfg::kDS;
        if (need_mask)
          bwd_softmax_half<true>(s, dp, stat_addr, scale_log2, row_valid ? kv_pos - q_pos : 32,
                                 tS + half * 32, tS + half * 32 + 16, ds_row_addr, half * 4, row);
        else
          bwd_softmax_half<false>(s, dp, stat_addr, scale_log2, 0, tS + half * 32,
                                  tS + half * 32 + 16, ds_row_addr, half * 4, row);
        fence_proxy_async_smem();
        tmem_st_wait();
        tc_fence_before();
        mbar_arrive(&bars->p_ready);
      }
      // item epilogue: dV (half 0) / dK (half 1) rows out of TMEM
      mbar_wait(&bars->dkv_full, m & 1);
      tc_fence_after();
      {
        const uint32_t tacc = tmem_base + lane_addr + (half == 0 ? Cfg::kColDV : Cfg::kColDK);
        const float f = half == 0 ? 1.f : scale;
        __nv_bfloat16* dst = reinterpret_cast<__nv_bfloat16*>(dst_b);
        if (!dkv_f32 && it.kv_rows == 128) {
          // Full bf16 tile: the accumulator rows leave TMEM first (dV / dK are free for the next
          // item at once), then go panel by panel (64 columns = 128 B per row) through this
          // warpgroup's dS^T buffer — idle between items — in the SWIZZLE_128B layout of the
          // dk / dv tensor map, one TMA store per panel.  A thread owns a row: direct stores touch
          // 32 lines per instruction and back the LSU up in front of the next item's loads.
          uint32_t acc[D / 32][32];
#pragma unroll
          for (int c = 0; c < D / 32; ++c) tmem_ld32(tacc + c * 32, acc[c]);
          tmem_ld_wait();
          tc_fence_before();
          mbar_arrive(&bars->dkv_free);
          const uint32_t stage = smem_u32(ds_smem) + half * Cfg::kDS;
          const uint32_t stage_row = stage + row * 128;
          const uint32_t swz = row & 7;
#pragma unroll
          for (int pn = 0; pn < Cfg::kPanels; ++pn) {
            if (pn > 0 && issuer) bulk_wait_read0();    // the previous panel has been read
            if (pn > 0) named_bar_sync(4 + half, 128);
#pragma unroll
            for (int ch = 0; ch < 8; ++ch) {
              const int e = (ch & 3) * 8;               // element inside the 32-column chunk
              const uint32_t* a = acc[pn * 2 + (ch >> 2)];
              sts128(stage_row + ((ch ^ swz) << 4),
                     pack_bf16(__uint_as_float(a[e + 0]) * f, __uint_as_float(a[e + 1]) * f),
                     pack_bf16(__uint_as_float(a[e + 2]) * f, __uint_as_float(a[e + 3]) * f),
                     pack_bf16(__uint_as_float(a[e + 4]) * f, __uint_as_float(a[e + 5]) * f),
                     pack_bf16(__uint_as_float(a[e + 6]) * f, __uint_as_float(a[e + 7]) * f));
            }
            fence_proxy_async_smem();
            named_bar_sync(4 + half, 128);
            if (issuer) {
              tma_store_3d(half == 0 ? &tmap_dv : &tmap_dk, stage, pn * 64, it.kv_head, it.kv_row0);
              bulk_commit();
            }
          }
          staged = true;
        } else {
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t acc[32];
            tmem_ld32(tacc + c * 32, acc);
            tmem_ld_wait();
            if (row_valid && dkv_f32) {
              float4* d4 = reinterpret_cast<float4*>(dst_b) + c * 8;
#pragma unroll
              for (int i = 0; i < 8; ++i)
                d4[i] = make_float4(__uint_as_float(acc[4 * i + 0]) * f, __uint_as_float(acc[4 * i + 1]) * f,
                                    __uint_as_float(acc[4 * i + 2]) * f, __uint_as_float(acc[4 * i + 3]) * f);
            } else if (row_valid) {
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                int4 pk;
                pk.x = pack_bf16(__uint_as_float(acc[8 * i + 0]) * f, __uint_as_float(acc[8 * i + 1]) * f);
                pk.y = pack_bf16(__uint_as_float(acc[8 * i + 2]) * f, __uint_as_float(acc[8 * i + 3]) * f);
                pk.z = pack_bf16(__uint_as_float(acc[8 * i + 4]) * f, __uint_as_float(acc[8 * i + 5]) * f);
                pk.w = pack_bf16(__uint_as_float(acc[8 * i + 6]) * f, __uint_as_float(acc[8 * i + 7]) * f);
                *reinterpret_cast<int4*>(dst + c * 32 + i * 8) = pk;
              }
            }
          }
          tc_fence_before();
          mbar_arrive(&bars->dkv_free);
        }
      }
      ++m;
    }
    if (issuer) bulk_wait0();                          // dk / dv stores of the last item
  } else {
    // ------------------------------------------------------------------ dQ drain (warps 12-15)
    reg_dealloc<Cfg::kRegsDrain>();
    const int drow = (warp & 3) * 32 + lane;           // d index = TMEM lane of dQ^T
    const uint32_t tDQ = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + Cfg::kColDQ;
    const uint32_t dq_addr = smem_u32(dq_smem) + drow * 4;
    const bool leader = role == 12 && lane == 0;
    uint32_t n = 0;
    for (int idx = item_begin; idx < item_end; ++idx) {
      const BwdItem it = items[idx];
      if (it.n_iters == 0) continue;
      for (IterWalk w(it, subs, G); !w.done(); w.next(), ++n) {
        mbar_wait(&bars->dq_full, n & 1);
        tc_fence_after();
        uint32_t acc[2][32];
        tmem_ld32(tDQ, acc[0]);
        tmem_ld32(tDQ + 32, acc[1]);
        tmem_ld_wait();
        tc_fence_before();
        mbar_arrive(&bars->dq_free);
        if (leader) bulk_wait_read0();                  // previous reduce has read the staging
        named_bar_sync(1, 128);
        if (drow < D) {
#pragma unroll
          for (int q = 0; q < FCP_BQ; ++q) sts32(dq_addr + q * D * 4, acc[q >> 5][q & 31]);
        }
        fence_proxy_async_smem();
        named_bar_sync(1, 128);
        if (leader) {
          const int head = it.kv_head * G + w.g;
          bulk_reduce_add_f32(dq_acc + ((int64_t)head * n_q_pad + w.pad_row()) * D, dq_smem,
                              (uint32_t)w.valid() * D * 4);
          bulk_commit();
        }
      }
    }
    if (leader) bulk_wait0();
  }

  tc_fence_before();
  __syncthreads();
  if (role == 1) {
    __syncwarp();
    tmem_dealloc<512>(tmem_base);
  }
}

template <int D>
int launch_bwd(const fcp_attn_args* a, const fcp_sched* s, const void* dO, void* dq, void* dk,
               void* dv) {
  using Cfg = BwdCfg<D>;
  cudaStream_t st = (cudaStream_t)a->stream;
  char* ws = static_cast<char*>(a->workspace);
  const int32_t* tile_meta = reinterpret_cast<const int32_t*>(ws + s->off_shard_meta);
  float2* lsed = reinterpret_cast<float2*>(ws + s->off_lsed);
  // dQ accumulates in fp32 across the KV tiles — and, with a caller-owned accumulator, across
  // the KV pieces of a local / prefix split (fcp.h section 2b)
  float* dq_acc = a->dq_accum ? a->dq_accum : reinterpret_cast<float*>(ws + s->off_dq);
  const bool keep = a->dq_accum && (a->dq_flags & FCP_DQ_KEEP);
  const bool convert = !(a->dq_accum && (a->dq_flags & FCP_DQ_NO_OUTPUT));
  const int n_pad_tiles = (int)(s->n_q_pad / FCP_BQ);

  if (n_pad_tiles > 0) {
    fcp_bwd_prep<D><<<dim3(n_pad_tiles, s->Hq), 256, 0, st>>>(
        static_cast<const __nv_bfloat16*>(a->o), static_cast<const __nv_bfloat16*>(dO), a->lse,
        tile_meta, lsed, keep ? nullptr : reinterpret_cast<float4*>(dq_acc), s->n_q, s->n_q_pad,
        s->Hq);
    if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
  }
  const int n_items = (int)s->bwd.size();
  if (n_items > 0) {
    CUtensorMap mq, mdo, mk, mv, mdk, mdv;
    if (!make_tmap_rows(&mq, a->q, D, s->Hq, s->n_q, FCP_BQ) ||
        !make_tmap_rows(&mdo, dO, D, s->Hq, s->n_q, FCP_BQ) ||
        !make_tmap_rows(&mk, a->k, D, s->Hkv, s->n_kv, 128) ||
        !make_tmap_rows(&mv, a->v, D, s->Hkv, s->n_kv, 128))
      return FCP_CUDA;
    // bf16 dk / dv leave through TMA stores; fp32 partials are stored row by row (maps unused)
    const bool f32 = a->dkv_dtype == FCP_DTYPE_F32;
    if (!make_tmap_rows(&mdk, f32 ? a->k : dk, D, s->Hkv, s->n_kv, 128) ||
        !make_tmap_rows(&mdv, f32 ? a->v : dv, D, s->Hkv, s->n_kv, 128))
      return FCP_CUDA;
    auto kern = fcp_attn_bwd_main<D>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             Cfg::kSmemBytes) != cudaSuccess)
      return FCP_CUDA;
    const int grid = s->n_cta;
    if (a->ev_start && cudaEventRecord((cudaEvent_t)a->ev_start, st) != cudaSuccess)
      return FCP_CUDA;
    kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, st>>>(
        mq, mdo, mk, mv, mdk, mdv, reinterpret_cast<const BwdItem*>(ws + s->off_bwd),
        reinterpret_cast<const int32_t*>(ws + s->off_bwd_cta),
        reinterpret_cast<const BwdSub*>(ws + s->off_sub), lsed, dq_acc, dk, dv,
        a->dkv_dtype == FCP_DTYPE_F32, s->n_q_pad, s->Hkv, s->G, a->scale, a->scale * kLog2e);
    if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
    if (a->ev_stop && cudaEventRecord((cudaEvent_t)a->ev_stop, st) != cudaSuccess)
      return FCP_CUDA;
  }
  if (n_pad_tiles > 0 && convert) {
    fcp_bwd_dq_convert<D><<<dim3(n_pad_tiles, s->Hq), 256, 0, st>>>(
        dq_acc, tile_meta, static_cast<__nv_bfloat16*>(dq), s->n_q_pad, s->Hq, a->scale);
    if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
  }
  return FCP_OK;
}

}  // namespace

extern "C" int fcp_attn_bwd(const fcp_attn_args* a, const void* dO, void* dq, void* dk, void* dv) {
  if (!a || !a->sched || !a->workspace || !a->q || !a->o || !a->lse || !dO) return FCP_INVALID_ARG;
  // k, v, dk, dv may be NULL when the schedule has no key at all (n_kv == 0)
  if (a->sched->n_kv > 0 && (!a->k || !a->v || !dk || !dv)) return FCP_INVALID_ARG;
  if (!dq && !(a->dq_accum && (a->dq_flags & FCP_DQ_NO_OUTPUT))) return FCP_INVALID_ARG;
  if (a->dq_accum && (reinterpret_cast<uintptr_t>(a->dq_accum) & 15)) return FCP_MISALIGNED;
  const fcp_sched* s = a->sched;
  if (a->dkv_dtype != FCP_DTYPE_BF16 && a->dkv_dtype != FCP_DTYPE_F32) return FCP_UNSUPPORTED;
  for (const void* p : {a->q, a->k, a->v, (const void*)a->o, (const void*)a->workspace, dO,
                        (const void*)dq, (const void*)dk, (const void*)dv})
    if (reinterpret_cast<uintptr_t>(p) & 15) return FCP_MISALIGNED;
  if (s->D == 128) return launch_bwd<128>(a, s, dO, dq, dk, dv);
  if (s->D == 64) return launch_bwd<64>(a, s, dO, dq, dk, dv);
  return FCP_UNSUPPORTED;
}

// ------------------------------------------------------------------------------------------
// fcp_attn_bwd_static: the backward on a workspace the library owns (fcp.h section 4).
// ------------------------------------------------------------------------------------------
namespace {
// Held by every GPU that loads the library, from module load to process exit; uninitialised
// (no bytes in the .so).  In host code this name is only a handle for cudaGetSymbolAddress:
// kernels get the device address that static_workspace() returns.
static __device__ __align__(256) unsigned char fcp_static_ws[FCP_STATIC_WORKSPACE_BYTES];

// Device address of fcp_static_ws on the CURRENT device, looked up once per device (each device
// has its own copy of the array at its own address) and kept in a write-once table behind
// atomics; nullptr when the lookup fails.
void* static_workspace() {
  constexpr int kMaxDev = 64;
  static std::atomic<void*> cache[kMaxDev];
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
  const bool cached = dev >= 0 && dev < kMaxDev;
  if (cached) {
    void* p = cache[dev].load(std::memory_order_acquire);
    if (p) return p;
  }
  void* p = nullptr;
  if (cudaGetSymbolAddress(&p, fcp_static_ws) != cudaSuccess || p == nullptr) return nullptr;
  if (cached) cache[dev].store(p, std::memory_order_release);
  return p;
}
}  // namespace

extern "C" int fcp_attn_bwd_static(const fcp_attn_args* a, const void* dO, void* dq, void* dk,
                                   void* dv) {
  if (!a || !a->sched || a->workspace) return FCP_INVALID_ARG;
  if (a->sched->total > (size_t)FCP_STATIC_WORKSPACE_BYTES) return FCP_TOO_LARGE;
  void* ws = static_workspace();
  if (!ws) {
    cudaGetLastError();
    return FCP_CUDA;
  }
  fcp_attn_args b = *a;
  b.workspace = ws;
  // the lists go first on the same stream: stream order puts them before the kernels, and
  // behind every earlier call that used the workspace on this stream
  const int st = fcp_sched_upload(a->sched, ws, a->stream);
  if (st != FCP_OK) return st;
  return fcp_attn_bwd(&b, dO, dq, dk, dv);
}
