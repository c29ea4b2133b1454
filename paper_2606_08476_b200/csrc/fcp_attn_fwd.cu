// Document-masked causal attention forward for sm_100a.
//
// One persistent CTA per SM.  A work item is one 128-row q tile of one shard for a pack of NQ
// query heads that share a kv head (GQA): the NQ tiles share every K/V tile staged in shared
// memory.  Per q tile t the chain is   S_t(j) -> softmax -> P_t(j) -> O_t += P_t(j) V_j ->
// S_t(j+1) = Q_t K_{j+1}^T -> ...   The bf16 P_t is written by the softmax threads over the
// first 64 TMEM columns of S_t (whose fp32 scores they hold in registers by then) and is the A
// operand of the PV product straight from TMEM, so that product reads only V from shared memory
// and no P ever crosses it.  The two tiles' chains alternate: while the tensor pipe works on
// tile t, the softmax of the other tile has the MUFU to itself (a named-barrier token keeps the
// two from exponentiating at the same time: two warps per sub-partition in lockstep idle the
// MUFU during their loads and stores).
//
//   warp 0      TMA producer   Q (once per item); K/V tiles through a 3-slot ring in the order
//                              the MMAs consume them: K0, V0, K1, V1, ...
//   warp 1      MMA issuer     one elected thread; per KV tile j and q tile t: O_t += P_t(j) V_j
//                              (A = P from TMEM, B = V MN-major), then S_t(j+1) (SS) — program
//                              order on the in-order tensor pipe is what protects P_t(j) from
//                              S_t(j+1)
//   warps 4..   softmax        one warpgroup per q tile, one query row per thread: mask from
//                              (q_pos0 + row, kv_len), online softmax in the log2 domain that
//                              exponentiates against the running max of the earlier tiles (no
//                              max -> exp dependency) and rescales O only when a row grew by
//                              more than 2^8; a quarter of the exponentials of that fast path
//                              run as a degree-3 polynomial on the FMA pipe (packed fp32x2),
//                              the rest on the MUFU; epilogue o = O / l
//
// TMEM columns: S_t at 128 t (P_t over its first 64), O_t at 128 (NQ + t).
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
#ifndef FCP_TOKEN_QUARTER
#define FCP_TOKEN_QUARTER 3
#endif
constexpr int kTokenQuarter = FCP_TOKEN_QUARTER;   // quarter of the exponential loop after which the MUFU token moves on
#ifndef FCP_POLY_MASK
#define FCP_POLY_MASK 0x55
#endif
// Of the 8 groups of 4 scores in a 32-column chunk, the groups whose bit is set here take 2 of
// their 4 exponentials from the FMA pipe instead of the MUFU (0x55 = a quarter of all ex2)
constexpr unsigned kPolyMask = FCP_POLY_MASK;
// 2^x for two values on the FMA pipe (packed fp32x2): x = n + f with f in [-0.5, 0.5] by the
// round-to-nearest magic constant, degree-3 polynomial for 2^f (max relative error 1.1e-4, well
// below the 2^-9 of the bf16 P it feeds), exponent added as an integer.  x >= -120.
__device__ __forceinline__ void exp2_fma(float x0, float x1, float& p0, float& p1) {
  const f32x2 x = pack2(x0, x1);
  const f32x2 t = add2(x, pack2(12582912.f, 12582912.f));            // 1.5 * 2^23
  const f32x2 f = fma2(add2(t, pack2(-12582912.f, -12582912.f)), pack2(-1.f, -1.f), x);
  f32x2 p = fma2(pack2(0.0555041086f, 0.0555041086f), f, pack2(0.2402265069f, 0.2402265069f));
  p = fma2(p, f, pack2(0.6931471806f, 0.6931471806f));
  p = fma2(p, f, pack2(1.0f, 1.0f));
  float t0, t1, q0, q1;
  unpack2(t, t0, t1);
  unpack2(p, q0, q1);
  p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
  p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}
constexpr float kRescaleThreshold = 8.0f;

// 3-D tiled store shared -> global through a tensor map (coordinates as tma_load_3d)
__device__ __forceinline__ void tma_store_3d(const void* tmap, const void* smem_src, int32_t c0,
                                             int32_t c1, int32_t c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::
                   "l"(tmap), "r"(smem_u32(smem_src)), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }   // log2 units: rescale O only when the max grew by > 2^8

template <int D, int NQ>
struct FwdCfg {
  static constexpr int kTileBytes = 128 * D * 2;           // one Q, K or V tile
  static constexpr int kPanelBytes = 128 * 128;            // 128 rows x 64 bf16
  static constexpr int kPanels = D / 64;
  static constexpr int kStages = (D == 128) ? 3 : 6;       // ring slots, each one K or V tile
  static constexpr int kThreads = 128 + 128 * NQ;
  static constexpr int kTmemCols = 256 * NQ;
  static constexpr int kOffRing = NQ * kTileBytes;
  static constexpr int kOffOut = kOffRing + kStages * kTileBytes;   // NQ staging tiles for o
  static constexpr int kSmemData = kOffOut + NQ * kTileBytes;
  static constexpr int kSmemBytes = 1024 + kSmemData + 256;
  // registers per thread after setmaxnreg (multiples of 8).  The CTA owns (launch registers x
  // threads): the sum over its warpgroups must stay below.
  static constexpr int kLaunchRegs = (65536 / kThreads) / 8 * 8 > 255 ? 248 : (65536 / kThreads) / 8 * 8;
  static constexpr int kRegsCtl = 72;
  static constexpr int kRegsSoftmaxRaw = (kLaunchRegs * (kThreads / 128) - kRegsCtl) / NQ / 8 * 8;
  static constexpr int kRegsSoftmax = kRegsSoftmaxRaw > 232 ? 232 : kRegsSoftmaxRaw;
};
static_assert(FwdCfg<128, 2>::kSmemBytes <= 232448, "fwd shared memory exceeds 227 KB");

struct FwdBarriers {
  uint64_t q_full, q_empty;
  uint64_t kv_full[8], kv_empty[8];
  uint64_t s_full[2];    // S_t written by the MMAs (and, in pipe order, the O_t += P_t V before
                         // it complete)                           -> softmax
  uint64_t p_ready[2];   // S_t in registers, bf16 P_t written over its first 64 TMEM columns,
                         // O_t rescaled                           -> MMA
  uint64_t pv_done[2];   // last O_t += P_t V of the item complete -> epilogue
  uint64_t o_empty[2];   // epilogue has read O_t                  -> MMA may overwrite O_t
  uint32_t tmem_base;
};
static_assert(sizeof(FwdBarriers) <= 256, "barrier block");

template <int D, int NQ>
__global__ void __launch_bounds__(FwdCfg<D, NQ>::kThreads, 1)
fcp_attn_fwd_kernel(const __grid_constant__ CUtensorMap tmap_q,
                    const __grid_constant__ CUtensorMap tmap_k,
                    const __grid_constant__ CUtensorMap tmap_v,
                    const __grid_constant__ CUtensorMap tmap_o,
                    const FwdItem* __restrict__ items, const int32_t* __restrict__ cta_off,
                    __nv_bfloat16* __restrict__ o, float* __restrict__ lse,
                    int64_t n_q, int Hq, float scale_log2) {
  using Cfg = FwdCfg<D, NQ>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) &
                                             ~uintptr_t(1023));
  uint8_t* q_smem = smem;                                  // NQ tiles
  uint8_t* ring = smem + Cfg::kOffRing;                    // kStages tiles
  uint8_t* out_smem = smem + Cfg::kOffOut;                 // NQ tiles: o rows staged for the TMA store
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
      mbar_init(&bars->pv_done[t], 1);
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

  if (warp < 4) {
    reg_dealloc<Cfg::kRegsCtl>();
    if (warp == 0 && lane == 0) {
      // ---------------------------------------------------------------- TMA producer
      prefetch_tmap(&tmap_q);
      prefetch_tmap(&tmap_k);
      prefetch_tmap(&tmap_v);
      uint32_t slot = 0, sph = 0, iph = 0;
      auto load_kv = [&](const CUtensorMap* tm, int kv_head, int row0) {
        mbar_wait(&bars->kv_empty[slot], sph ^ 1);
        mbar_arrive_expect_tx(&bars->kv_full[slot], Cfg::kTileBytes);
        for (int pn = 0; pn < Cfg::kPanels; ++pn)
          tma_load_3d(ring + slot * Cfg::kTileBytes + pn * Cfg::kPanelBytes, tm,
                      &bars->kv_full[slot], pn * 64, kv_head, row0);
        if (++slot == (uint32_t)Cfg::kStages) { slot = 0; sph ^= 1; }
      };
      for (int idx = item_begin; idx < item_end; ++idx) {
        const FwdItem it = items[idx];
        const int n = it.n_kv_tiles;
        if (n == 0) continue;
        mbar_wait(&bars->q_empty, iph ^ 1);
        mbar_arrive_expect_tx(&bars->q_full, NQ * Cfg::kTileBytes);
        for (int t = 0; t < NQ; ++t)
          for (int pn = 0; pn < Cfg::kPanels; ++pn)
            tma_load_3d(q_smem + t * Cfg::kTileBytes + pn * Cfg::kPanelBytes, &tmap_q,
                        &bars->q_full, pn * 64, it.head0 + t, it.q_row0);
        // consumption order of the MMAs: K0, then per tile j: V_j, K_{j+1}
        load_kv(&tmap_k, it.kv_head, it.kv_row0);
        for (int j = 0; j < n; ++j) {
          load_kv(&tmap_v, it.kv_head, it.kv_row0 + j * FCP_TK);
          if (j + 1 < n) load_kv(&tmap_k, it.kv_head, it.kv_row0 + (j + 1) * FCP_TK);
        }
        iph ^= 1;
      }
    } else if (warp == 1 && elect_one()) {
      // ---------------------------------------------------------------- MMA issuer
      // One elected thread.  Per q tile t the chain is
      //   S_t(0) | per KV tile j:  O_t += P_t(j) V_j  then  S_t(j+1) = Q_t K_{j+1}^T
      // with the two tiles' chains interleaved.  P_t is the A operand straight from TMEM: the
      // softmax warpgroup writes it (bf16) over the first 64 columns of S_t once S_t sits in
      // registers, so S_t(j+1) must follow O_t += P_t(j) V_j in the (in-order) tensor pipe — which
      // this issue order gives without a barrier — and the PV product reads only V from shared
      // memory.  While tile t waits for its next S the other tile's softmax has the MUFU alone.
      constexpr uint32_t idesc_qk = umma_idesc_bf16(128, 128, 0, 0);
      constexpr uint32_t idesc_pv = umma_idesc_bf16(128, D, 0, 1);
      constexpr int kSteps = D / 16;
      constexpr uint32_t kHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO, version, swizzle
      constexpr uint32_t kTileStep = Cfg::kTileBytes >> 4;
      auto lo_word = [](uint32_t saddr, uint32_t lbo) { return ((saddr & 0x3FFFF) >> 4) | ((lbo >> 4) << 16); };
      auto desc = [](uint32_t lo) { return ((uint64_t)kHi << 32) | lo; };
      const uint32_t q_kmaj = lo_word(smem_u32(q_smem), 16);                     // A of S (tile 0)
      const uint32_t ring_kmaj = lo_word(smem_u32(ring), 16);                    // K tile, slot 0
      const uint32_t ring_mnmaj = lo_word(smem_u32(ring), Cfg::kPanelBytes);     // V tile, slot 0

      auto issue_qk = [&](int t, uint32_t kslot) {
        const uint32_t a0 = q_kmaj + t * kTileStep, b0 = ring_kmaj + kslot * kTileStep;
#pragma unroll
        for (int kk = 0; kk < kSteps; ++kk) {
          const uint32_t off = ((kk >> 2) * Cfg::kPanelBytes + (kk & 3) * 32) >> 4;
          umma_ss(tmem_base + t * 128, desc(a0 + off), desc(b0 + off), idesc_qk, kk > 0);
        }
      };
      // A = P_t from TMEM: 16 keys of bf16 = 8 columns per K step
      auto issue_pv = [&](int t, uint32_t vslot, bool acc) {
        const uint32_t b0 = ring_mnmaj + vslot * kTileStep;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          umma_ts(tmem_base + (NQ + t) * 128, tmem_base + t * 128 + kk * 8,
                  desc(b0 + kk * (2048 >> 4)), idesc_pv, (acc || kk > 0) ? 1u : 0u);
      };
      auto ring_next = [](uint32_t& s_, uint32_t& p_) {
        if (++s_ == (uint32_t)Cfg::kStages) { s_ = 0; p_ ^= 1; }
      };

      uint32_t slot = 0, sph = 0;      // ring position / phase parity of the next tile to consume
      uint32_t ppp = 0;                // parity of p_ready (both tiles advance together)
      uint32_t iph = 0;                // item parity (q_full; o_empty of the previous item)

      for (int idx = item_begin; idx < item_end; ++idx) {
        const int n = items[idx].n_kv_tiles;
        if (n == 0) continue;
        mbar_wait(&bars->q_full, iph);
        mbar_wait(&bars->kv_full[slot], sph);
        tc_fence_after();
#pragma unroll
        for (int t = 0; t < NQ; ++t) {
          // S_t is free: the previous item's last P_t V was issued before (in-order pipe)
          issue_qk(t, slot);
          umma_commit(&bars->s_full[t]);
        }
        umma_commit(&bars->kv_empty[slot]);
        if (n == 1) umma_commit(&bars->q_empty);
        ring_next(slot, sph);
        for (int j = 0; j < n; ++j) {
          const bool has_next = j + 1 < n;
          const uint32_t vslot = slot, vph = sph;
          uint32_t kslot = slot, kph = sph;
          ring_next(kslot, kph);                    // K_{j+1} follows V_j in the ring
#pragma unroll
          for (int t = 0; t < NQ; ++t) {
            if (t == 0) mbar_wait(&bars->kv_full[vslot], vph);
            if (j == 0) mbar_wait(&bars->o_empty[t], iph ^ 1);
            mbar_wait(&bars->p_ready[t], ppp);
            tc_fence_after();
            issue_pv(t, vslot, j > 0);
            if (!has_next) umma_commit(&bars->pv_done[t]);
            if (t == NQ - 1) umma_commit(&bars->kv_empty[vslot]);   // V_j: both tiles have read it
            if (has_next) {
              if (t == 0) {
                mbar_wait(&bars->kv_full[kslot], kph);
                tc_fence_after();
              }
              issue_qk(t, kslot);
              umma_commit(&bars->s_full[t]);
            }
          }
          ppp ^= 1;
          ring_next(slot, sph);
          if (has_next) {
            umma_commit(&bars->kv_empty[kslot]);
            if (j + 2 == n) umma_commit(&bars->q_empty);
            ring_next(slot, sph);
          }
        }
        iph ^= 1;
      }
    }
  } else {
    // ------------------------------------------------------------------ softmax + epilogue
    // One warpgroup per q tile, one query row per thread (TMEM lane = row).  Online softmax in
    // the log2 domain, per KV tile:
    //   fast path  p = exp2(s c - m) against the running max m of the earlier tiles while the
    //              tile max is computed on the side (no max -> exp dependency); kept when no
    //              row of the warp exceeds m by more than 2^kRescaleThreshold;
    //   exact path (first tile of a row, or a row grew): tile max first, m, l and O rescaled —
    //              S stays in registers until the path is chosen, so nothing is approximated.
    // S is released to the MMA thread as soon as it sits in registers; P goes to shared memory
    // after the previous O_t += P V has finished reading it.
    reg_alloc<Cfg::kRegsSoftmax>();
    const int t = (warp >> 2) - 1;                 // q tile of this warpgroup
    const int row = (warp & 3) * 32 + lane;        // query row = TMEM lane
    const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem_base + lane_addr + t * 128;
    const uint32_t tO = tmem_base + lane_addr + (NQ + t) * 128;
    uint32_t s_ph = 0, pv_ph = 0;
    if (NQ == 2 && t == 1) named_bar_arrive(2, 256);        // tile 0 holds the MUFU token first
    const bool o_al32 = (reinterpret_cast<uintptr_t>(o) & 31) == 0;
    FwdItem nxt;
    if (item_begin < item_end) nxt = items[item_begin];

    for (int idx = item_begin; idx < item_end; ++idx) {
      const FwdItem it = nxt;
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
        if (idx + 1 < item_end) nxt = items[idx + 1];
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
        // MUFU token: the exponentials of the two q tiles take turns (16 ex2/clk/SM bound a tile
        // at 1024 clocks; in lockstep both warpgroups would do their loads, waits and stores at
        // the same time and leave the MUFU idle meanwhile)
        if (NQ == 2) named_bar_sync(2 + t, 256);
        if (NQ == 2 && kTokenQuarter < 0) named_bar_arrive(2 + (t ^ 1), 256);
        uint32_t pk[64];
        float alpha = 1.f;
        bool any_grow = false;
        const f32x2 scale2 = pack2(scale_log2, scale_log2);
        // p = exp2(s c - m_ref) for the whole row, packed to bf16; returns the row sum.  Packed
        // fp32x2 FMA / ADD and the 3-input max keep the loop MUFU-bound (6 issue slots per 2
        // elements of which 2 are MUFU).
        bool token_passed = NQ != 2 || kTokenQuarter < 0;
        auto exp_row = [&](float m_ref, float& mx_out, bool with_max) -> float {
          const f32x2 negm2 = pack2(-m_ref, -m_ref);
          f32x2 sum_a = pack2(0.f, 0.f), sum_b = sum_a;
          float mx_a = -INFINITY, mx_b = -INFINITY;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
              const float s0 = __uint_as_float(sr[c][2 * i]), s1 = __uint_as_float(sr[c][2 * i + 1]);
              const float s2 = __uint_as_float(sr[c][2 * i + 2]), s3 = __uint_as_float(sr[c][2 * i + 3]);
              if (with_max) {
                mx_a = max3(mx_a, s0, s1);
                mx_b = max3(mx_b, s2, s3);
              }
              float x0, x1, x2, x3;
              unpack2(fma2(pack2(s0, s1), scale2, negm2), x0, x1);
              unpack2(fma2(pack2(s2, s3), scale2, negm2), x2, x3);
              const float p0 = fast_exp2(x0), p1 = fast_exp2(x1);
              float p2, p3;
              // fast path only: every row of the warp has a finite running max there, so a masked
              // score may come out as 2^-120 instead of 0 without changing l or O
              if (with_max && ((kPolyMask >> (i >> 1)) & 1u)) {
                exp2_fma(fmaxf(x2, -120.f), fmaxf(x3, -120.f), p2, p3);
              } else {
                p2 = fast_exp2(x2);
                p3 = fast_exp2(x3);
              }
              sum_a = add2(sum_a, pack2(p0, p1));
              sum_b = add2(sum_b, pack2(p2, p3));
              pk[c * 16 + i] = pack_bf16(p0, p1);
              pk[c * 16 + i + 1] = pack_bf16(p2, p3);
            }
            // this quarter of the P row (32 keys = 16 bf16 pairs) goes over the first columns of
            // S_t — the whole of S_t is in registers, and the previous O_t += P V finished before
            // S_t was written (same pipe, issued earlier)
            tmem_st16(tS + c * 16, *reinterpret_cast<const uint32_t(*)[16]>(&pk[c * 16]));
            // hand the MUFU token on part-way: the other tile starts its exponentials while
            // this one finishes (two warps per sub-partition keep the MUFU saturated; one alone
            // is latency-bound)
            if (c == kTokenQuarter && !token_passed) {
              named_bar_arrive(2 + (t ^ 1), 256);
              token_passed = true;
            }
          }
          mx_out = fmaxf(mx_a, mx_b);
          float lo, hi;
          unpack2(add2(sum_a, sum_b), lo, hi);
          return lo + hi;
        };
        bool exact = j == 0 || __any_sync(0xffffffffu, m == -INFINITY);
        if (!exact) {
          // ---- fast path: running max of the earlier tiles, tile max on the side
          float mx;
          const float sum = exp_row(m, mx, true);
          exact = __any_sync(0xffffffffu, mx * scale_log2 > m + kRescaleThreshold);
          if (!exact) l += sum;
        }
        if (exact) {
          // ---- exact path (first tile of a row, or a row grew): tile max first
          float mx_a = -INFINITY, mx_b = -INFINITY;
#pragma unroll
          for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int i = 0; i < 32; i += 4) {
              mx_a = max3(mx_a, __uint_as_float(sr[c][i]), __uint_as_float(sr[c][i + 1]));
              mx_b = max3(mx_b, __uint_as_float(sr[c][i + 2]), __uint_as_float(sr[c][i + 3]));
            }
          const float m_new = fmaxf(m, fmaxf(mx_a, mx_b) * scale_log2);
          const bool grow = m_new > m + kRescaleThreshold;   // also first finite max (m = -inf)
          any_grow = __any_sync(0xffffffffu, grow);
          if (grow) {
            alpha = fast_exp2(m - m_new);                   // m = -inf -> 0
            m = m_new;
          }
          float unused;
          const float sum = exp_row((m == -INFINITY) ? 0.f : m, unused, false);
          l = l * alpha + sum;
        }
        if (any_grow && j > 0) {                            // rescale the running O row
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
      mbar_wait(&bars->pv_done[t], pv_ph);
      pv_ph ^= 1;
      tc_fence_after();
      const float inv = l > 0.f ? 1.f / l : 0.f;
      // The whole O row leaves TMEM first: O_t is free for the next item's first PV product at
      // once, and the loads do not queue behind the store burst below.
      uint32_t orow[D / 32][32];
#pragma unroll
      for (int c = 0; c < D / 32; ++c) tmem_ld32(tO + c * 32, orow[c]);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(&bars->o_empty[t]);
      // next item's descriptor: issued before the stores so that it does not wait behind them
      if (idx + 1 < item_end) nxt = items[idx + 1];
      if (it.q_rows == FCP_TQ) {
        // Full tile: rows are staged in shared memory in the SWIZZLE_128B layout of the o tensor
        // map and leave with one TMA store per 64-column panel (a thread owns a row, so direct
        // stores would touch 32 lines per instruction and back up the LSU for ~2000 clocks).
        const bool issuer = (warp & 3) == 0 && lane == 0;
        if (issuer) bulk_wait_read0();                 // the previous item's store has read the tile
        named_bar_sync(4 + t, 128);
        const uint32_t out_row = smem_u32(out_smem) + t * Cfg::kTileBytes + row * 128;
        const uint32_t swz = row & 7;
#pragma unroll
        for (int c = 0; c < D / 32; ++c)
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int ch = c * 4 + i;                  // 16-byte chunk of the row
            sts128(out_row + (ch >> 3) * Cfg::kPanelBytes + (((ch & 7) ^ swz) << 4),
                   pack_bf16(__uint_as_float(orow[c][8 * i + 0]) * inv, __uint_as_float(orow[c][8 * i + 1]) * inv),
                   pack_bf16(__uint_as_float(orow[c][8 * i + 2]) * inv, __uint_as_float(orow[c][8 * i + 3]) * inv),
                   pack_bf16(__uint_as_float(orow[c][8 * i + 4]) * inv, __uint_as_float(orow[c][8 * i + 5]) * inv),
                   pack_bf16(__uint_as_float(orow[c][8 * i + 6]) * inv, __uint_as_float(orow[c][8 * i + 7]) * inv));
          }
        fence_proxy_async_smem();
        named_bar_sync(4 + t, 128);
        if (issuer) {
#pragma unroll
          for (int pn = 0; pn < Cfg::kPanels; ++pn)
            tma_store_3d(&tmap_o, out_smem + t * Cfg::kTileBytes + pn * Cfg::kPanelBytes, pn * 64,
                         head, it.q_row0);
          bulk_commit();
        }
      } else if (row_valid) {
        // ragged last tile of a shard: the rows after it belong to another shard, so each thread
        // stores its own row (32-byte stores when o is 32-byte aligned)
#pragma unroll
        for (int c = 0; c < D / 32; ++c)
#pragma unroll
          for (int i = 0; i < 2; ++i) {
            uint32_t w[8];
#pragma unroll
            for (int k = 0; k < 8; ++k)
              w[k] = pack_bf16(__uint_as_float(orow[c][16 * i + 2 * k]) * inv,
                               __uint_as_float(orow[c][16 * i + 2 * k + 1]) * inv);
            __nv_bfloat16* dst = o_row + c * 32 + i * 16;
            if (o_al32) {
              stg256(dst, w);
            } else {
              *reinterpret_cast<int4*>(dst) = make_int4(w[0], w[1], w[2], w[3]);
              *reinterpret_cast<int4*>(dst + 8) = make_int4(w[4], w[5], w[6], w[7]);
            }
          }
      }
      if (row_valid) *lse_row = l > 0.f ? kLn2 * (m + __log2f(l)) : -INFINITY;
    }
    if (NQ == 2 && t == 0) named_bar_sync(2, 256);          // consume tile 1's last token
    if ((warp & 3) == 0 && lane == 0) bulk_wait0();         // o stores of the last item
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
  CUtensorMap mq, mk, mv, mo;
  // an empty KV buffer (n_kv == 0: a PREFIX piece of shards that all start their document) has
  // no tile to load; its maps only need a valid base
  const void* kb = s->n_kv > 0 ? a->k : a->q;
  const void* vb = s->n_kv > 0 ? a->v : a->q;
  if (!make_tmap_rows(&mq, a->q, D, s->Hq, s->n_q, 128) ||
      !make_tmap_rows(&mk, kb, D, s->Hkv, s->n_kv, 128) ||
      !make_tmap_rows(&mv, vb, D, s->Hkv, s->n_kv, 128) ||
      !make_tmap_rows(&mo, a->o, D, s->Hq, s->n_q, 128))
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
      mq, mk, mv, mo, items,
      reinterpret_cast<const int32_t*>(static_cast<const char*>(a->workspace) + s->off_fwd_cta),
      static_cast<__nv_bfloat16*>(a->o), a->lse, s->n_q, s->Hq, a->scale * kLog2e);
  if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
  if (a->ev_stop && cudaEventRecord((cudaEvent_t)a->ev_stop, st) != cudaSuccess) return FCP_CUDA;
  return FCP_OK;
}

}  // namespace

extern "C" int fcp_attn_fwd(const fcp_attn_args* a) {
  if (!a || !a->sched || !a->workspace || !a->q || !a->o || !a->lse) return FCP_INVALID_ARG;
  const fcp_sched* s = a->sched;
  if (s->n_kv > 0 && (!a->k || !a->v)) return FCP_INVALID_ARG;   // k, v may be NULL when n_kv == 0
  for (const void* p : {a->q, a->k, a->v, (const void*)a->o, (const void*)a->workspace})
    if (reinterpret_cast<uintptr_t>(p) & 15) return FCP_MISALIGNED;
  if (s->fwd.empty()) return FCP_OK;
  if (s->D == 128) return s->NQ == 2 ? launch_fwd<128, 2>(a, s) : launch_fwd<128, 1>(a, s);
  if (s->D == 64) return s->NQ == 2 ? launch_fwd<64, 2>(a, s) : launch_fwd<64, 1>(a, s);
  return FCP_UNSUPPORTED;
}
