// Memory-bound device entry points of libfcp: sharding-aware KV gather,
// partial-result merge and the schedule upload.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>

#include "fcp_internal.h"
#include "fcp_sm100.cuh"

namespace {

// ------------------------------------------------------------------------------------------
// KV gather: a handful of contiguous row ranges of K and V are copied into k_out / v_out.
// Everything is expressed in 16-byte chunks; the destination is cut in 32 KB slabs that the
// CTAs take round-robin.  One thread per CTA drives the copy engine: cp.async.bulk global ->
// shared (mbarrier complete_tx) through a 3-slot ring, then cp.async.bulk shared -> global, so
// that 64 KB of loads per CTA (two CTAs per SM) are in flight with no register staging.
// HBM-bound: 2 tensors x (read + write) x rows x Hkv*D*2 bytes.
// ------------------------------------------------------------------------------------------
constexpr int kMaxRanges = 120;
constexpr int kSlab = 2048;                 // chunks per slab = 32 KB
constexpr int kGatherStages = 3;
constexpr int kGatherSmem = kGatherStages * kSlab * 16 + 64;

struct GatherRanges {
  int32_t n;
  int32_t pad;
  int64_t dst0[kMaxRanges + 1];   // first destination chunk of each range; dst0[n] = total
  int64_t src0[kMaxRanges];       // first source chunk of each range
};

__global__ void __launch_bounds__(32)
fcp_kv_gather_kernel(const int4* __restrict__ K, const int4* __restrict__ V,
                     int4* __restrict__ k_out, int4* __restrict__ v_out,
                     const __grid_constant__ GatherRanges rg) {
  extern __shared__ __align__(128) uint8_t gsm[];
  uint64_t* full = reinterpret_cast<uint64_t*>(gsm + kGatherStages * kSlab * 16);
  if (threadIdx.x != 0) return;
  using namespace fcp;
  for (int i = 0; i < kGatherStages; ++i) mbar_init(&full[i], 1);
  fence_barrier_init();
  const int64_t total = rg.dst0[rg.n];
  const int64_t n_slabs = (total + kSlab - 1) / kSlab;
  const int64_t n_work = 2 * n_slabs;                       // K slabs then V slabs
  const int64_t n_mine = blockIdx.x < n_work ? (n_work - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;

  // issue the loads of my w-th slab into ring slot w % kGatherStages
  auto load = [&](int64_t w) {
    const int64_t slab = blockIdx.x + w * gridDim.x;
    const bool is_v = slab >= n_slabs;
    const int64_t c0 = (is_v ? slab - n_slabs : slab) * kSlab;
    const int64_t c1 = c0 + kSlab < total ? c0 + kSlab : total;
    const int4* __restrict__ src = is_v ? V : K;
    const int st = (int)(w % kGatherStages);
    uint8_t* dst = gsm + st * kSlab * 16;
    mbar_arrive_expect_tx(&full[st], (uint32_t)(c1 - c0) * 16);
    int lo = 0, hi = rg.n - 1;                              // range that holds chunk c0
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (rg.dst0[mid] <= c0) lo = mid; else hi = mid - 1;
    }
    for (int64_t c = c0; c < c1; ++lo) {                    // a slab may straddle range borders
      const int64_t e = rg.dst0[lo + 1] < c1 ? rg.dst0[lo + 1] : c1;
      if (e > c) {
        bulk_load_1d(dst + (c - c0) * 16, src + rg.src0[lo] + (c - rg.dst0[lo]), (uint32_t)(e - c) * 16,
                     &full[st]);
        c = e;
      }
    }
  };
  const int64_t ahead = kGatherStages - 1;
  for (int64_t w = 0; w < ahead && w < n_mine; ++w) load(w);
  for (int64_t w = 0; w < n_mine; ++w) {
    const int64_t slab = blockIdx.x + w * gridDim.x;
    const bool is_v = slab >= n_slabs;
    const int64_t c0 = (is_v ? slab - n_slabs : slab) * kSlab;
    const int64_t c1 = c0 + kSlab < total ? c0 + kSlab : total;
    const int st = (int)(w % kGatherStages);
    if (w + ahead < n_mine) {
      // slot (w + ahead) % stages was read by the store of slab w - 1: wait for that read
      asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
      load(w + ahead);
    }
    mbar_wait(&full[st], (uint32_t)((w / kGatherStages) & 1));
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(
                     (is_v ? v_out : k_out) + c0),
                 "r"(smem_u32(gsm + st * kSlab * 16)), "r"((uint32_t)(c1 - c0) * 16)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  }
  asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------
// Merge: one sub-warp of D/8 lanes per (row, head); the group's first lane computes the two
// weights from the log-sum-exps and broadcasts them with a warp shuffle.
// ------------------------------------------------------------------------------------------
template <typename T> struct Vec8;
template <> struct Vec8<__nv_bfloat16> {
  static __device__ void load(const void* base, int64_t idx8, float (&f)[8]) {
    const int4 raw = reinterpret_cast<const int4*>(base)[idx8];
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&raw);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 x = __bfloat1622float2(h[i]);
      f[2 * i] = x.x;  f[2 * i + 1] = x.y;
    }
  }
  static __device__ void store(void* base, int64_t idx8, const float (&f)[8]) {
    int4 raw;
    __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&raw);
#pragma unroll
    for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
    reinterpret_cast<int4*>(base)[idx8] = raw;
  }
};
template <> struct Vec8<float> {
  static __device__ void load(const void* base, int64_t idx8, float (&f)[8]) {
    const float4 a = reinterpret_cast<const float4*>(base)[2 * idx8];
    const float4 b = reinterpret_cast<const float4*>(base)[2 * idx8 + 1];
    f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w; f[4] = b.x; f[5] = b.y; f[6] = b.z; f[7] = b.w;
  }
  static __device__ void store(void* base, int64_t idx8, const float (&f)[8]) {
    reinterpret_cast<float4*>(base)[2 * idx8] = make_float4(f[0], f[1], f[2], f[3]);
    reinterpret_cast<float4*>(base)[2 * idx8 + 1] = make_float4(f[4], f[5], f[6], f[7]);
  }
};

// ------------------------------------------------------------------------------------------
// dKV scatter-add: the inverse of the gather.  dst (fp32, global token order) += src (bf16 or
// fp32, gathered order) over the same contiguous ranges.  HBM-bound read-modify-write: per
// element 2 or 4 B read + 4 B read + 4 B write.  One thread handles 8 consecutive elements
// (16 B of bf16 / 32 B of fp32 in, 32 B in and out of the accumulator); all loads of a thread's
// kScatterUnroll chunks are issued before its stores.
// ------------------------------------------------------------------------------------------
constexpr int kScatterThreads = 256;
constexpr int kScatterUnroll = 4;

template <typename T>
__global__ void __launch_bounds__(kScatterThreads)
fcp_kv_scatter_add_kernel(const T* __restrict__ dk_r, const T* __restrict__ dv_r,
                          float* __restrict__ dK, float* __restrict__ dV,
                          const __grid_constant__ GatherRanges rg) {
  // rg is expressed in units of 8 elements: dst0 = offsets in the rank buffer, src0 = in dK/dV
  const int64_t total = rg.dst0[rg.n];
  constexpr int64_t kSpan = (int64_t)kScatterThreads * kScatterUnroll;
  const int64_t n_spans = (total + kSpan - 1) / kSpan;
  for (int64_t span = blockIdx.x; span < 2 * n_spans; span += gridDim.x) {
    const bool is_v = span >= n_spans;
    const int64_t c0 = (is_v ? span - n_spans : span) * kSpan;
    const T* __restrict__ src = is_v ? dv_r : dk_r;
    float* __restrict__ dst = is_v ? dV : dK;
    int lo = 0, hi = rg.n - 1;                              // range that holds unit c0
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (rg.dst0[mid] <= c0) lo = mid; else hi = mid - 1;
    }
    float in[kScatterUnroll][8];
    float4 acc[kScatterUnroll][2];
    float4* where[kScatterUnroll];
    int r = lo;
#pragma unroll
    for (int u = 0; u < kScatterUnroll; ++u) {
      const int64_t c = c0 + u * kScatterThreads + threadIdx.x;
      where[u] = nullptr;
      if (c < total) {
        while (c >= rg.dst0[r + 1]) ++r;
        Vec8<T>::load(src, c, in[u]);
        where[u] = reinterpret_cast<float4*>(dst) + 2 * (rg.src0[r] + (c - rg.dst0[r]));
        acc[u][0] = where[u][0];
        acc[u][1] = where[u][1];
      }
    }
#pragma unroll
    for (int u = 0; u < kScatterUnroll; ++u)
      if (where[u]) {
        where[u][0] = make_float4(acc[u][0].x + in[u][0], acc[u][0].y + in[u][1],
                                  acc[u][0].z + in[u][2], acc[u][0].w + in[u][3]);
        where[u][1] = make_float4(acc[u][1].x + in[u][4], acc[u][1].y + in[u][5],
                                  acc[u][1].z + in[u][6], acc[u][1].w + in[u][7]);
      }
  }
}

// fp32 -> bf16 (round to nearest even) of the reduced dK, dV: 8 elements per thread and step,
// 32 B in, 16 B out; blockIdx.y selects the tensor.  HBM-bound: 6 bytes per element.
__global__ void __launch_bounds__(256)
fcp_kv_reduce_finish_kernel(const float4* __restrict__ a, const float4* __restrict__ b,
                            int4* __restrict__ a_out, int4* __restrict__ b_out, int64_t n8) {
  const float4* __restrict__ src = blockIdx.y ? b : a;
  int4* __restrict__ dst = blockIdx.y ? b_out : a_out;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8;
       i += (int64_t)gridDim.x * blockDim.x) {
    const float4 x = src[2 * i], y = src[2 * i + 1];
    dst[i] = make_int4(fcp::pack_bf16(x.x, x.y), fcp::pack_bf16(x.z, x.w), fcp::pack_bf16(y.x, y.y),
                       fcp::pack_bf16(y.z, y.w));
  }
}

template <typename T>
__global__ void __launch_bounds__(256)
fcp_merge_kernel(const void* __restrict__ o_a, const float* __restrict__ lse_a,
                 const void* __restrict__ o_b, const float* __restrict__ lse_b,
                 void* o_out, float* lse_out, int64_t n_rows, int n_heads, int head_dim) {
  const int lanes = head_dim / 8;                       // lanes per (row, head): 8 or 16
  const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t pair = gid / lanes;                     // = row * n_heads + head
  const int sub = (int)(gid % lanes);
  const bool active = pair < n_rows * n_heads;
  float wa = 0.f, wb = 0.f;
  if (active && sub == 0) {
    const int64_t row = pair / n_heads, head = pair % n_heads;
    const float la = lse_a[head * n_rows + row], lb = lse_b[head * n_rows + row];
    const float m = fmaxf(la, lb);
    float lse = -INFINITY;
    if (m > -INFINITY) {                                 // guard (-inf) - (-inf)
      const float ea = __expf(la - m), eb = __expf(lb - m);
      const float z = ea + eb;
      wa = ea / z;  wb = eb / z;
      lse = m + __logf(z);
    }
    lse_out[head * n_rows + row] = lse;
  }
  const int src_lane = (threadIdx.x & 31) / lanes * lanes;
  wa = __shfl_sync(0xffffffffu, wa, src_lane);
  wb = __shfl_sync(0xffffffffu, wb, src_lane);
  if (!active) return;
  float a[8], b[8], r[8];
  Vec8<T>::load(o_a, gid, a);
  Vec8<T>::load(o_b, gid, b);
#pragma unroll
  for (int i = 0; i < 8; ++i) r[i] = wa * a[i] + wb * b[i];
  Vec8<T>::store(o_out, gid, r);
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }
bool valid_piece(int32_t piece) {
  return piece == FCP_PIECE_FULL || piece == FCP_PIECE_LOCAL || piece == FCP_PIECE_PREFIX;
}

}  // namespace

extern "C" int fcp_kv_gather(const fcp_plan* plan, int32_t rank, const void* K, const void* V,
                             void* k_out, void* v_out, int32_t n_kv_heads, int32_t head_dim,
                             void* stream, fcp_gather_counts* counts) {
  return fcp_kv_gather_piece(plan, rank, FCP_PIECE_FULL, K, V, k_out, v_out, n_kv_heads, head_dim,
                             stream, counts);
}

extern "C" int fcp_kv_gather_piece(const fcp_plan* plan, int32_t rank, int32_t piece, const void* K,
                                   const void* V, void* k_out, void* v_out, int32_t n_kv_heads,
                                   int32_t head_dim, void* stream, fcp_gather_counts* counts) {
  if (!plan || rank < 0 || rank >= plan->n_ranks || !valid_piece(piece) || !K || !V ||
      n_kv_heads < 1 || head_dim < 1)
    return FCP_INVALID_ARG;
  const int64_t row_bytes = (int64_t)n_kv_heads * head_dim * 2;
  if (row_bytes % 16 != 0) return FCP_UNSUPPORTED;
  if (!aligned16(K) || !aligned16(V) || !aligned16(k_out) || !aligned16(v_out))
    return FCP_MISALIGNED;
  RankView v;
  std::vector<int64_t> src, len;
  // merge ranges that are contiguous in the source (neighbouring documents held whole)
  const int st = fcp_guard([&] {
    fcp_build_rank_view(*plan, rank, v, piece);
    for (size_t g = 0; g < v.kv_len.size(); ++g) {
      if (v.kv_len[g] == 0) continue;
      if (!src.empty() && src.back() + len.back() == v.kv_src_start[g]) {
        len.back() += v.kv_len[g];
      } else {
        src.push_back(v.kv_src_start[g]);
        len.push_back(v.kv_len[g]);
      }
    }
    return (int)FCP_OK;
  });
  if (st != FCP_OK) return st;
  if (v.n_kv > 0 && (!k_out || !v_out)) return FCP_INVALID_ARG;   // an empty piece needs no buffer
  if (counts) {
    counts->total_tokens = v.n_kv;
    counts->remote_tokens = v.remote;
    counts->total_bytes = 2 * v.n_kv * row_bytes;
    counts->remote_bytes = 2 * v.remote * row_bytes;
    counts->n_ranges = (int32_t)src.size();
    counts->reserved = 0;
  }
  const int64_t cpr = row_bytes / 16;          // chunks per row
  const int num_sms = fcp_sm_count();
  // opt-in to > 48 KB of dynamic shared memory: a per-device (context) attribute, set on every
  // call so that a process driving several GPUs is served on each
  if (!src.empty() &&
      cudaFuncSetAttribute(fcp_kv_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           kGatherSmem) != cudaSuccess)
    return FCP_CUDA;
  int64_t dst_row = 0;
  for (size_t base = 0; base < src.size(); base += kMaxRanges) {
    GatherRanges rg;
    std::memset(&rg, 0, sizeof(rg));
    rg.n = (int32_t)std::min<size_t>(kMaxRanges, src.size() - base);
    int64_t c = 0;
    for (int i = 0; i < rg.n; ++i) {
      rg.dst0[i] = c;
      rg.src0[i] = src[base + i] * cpr;
      c += len[base + i] * cpr;
    }
    rg.dst0[rg.n] = c;
    const int64_t slabs = 2 * ((c + kSlab - 1) / kSlab);
    if (slabs == 0) continue;
    const int grid = (int)std::min<int64_t>(slabs, (int64_t)num_sms * 2);
    fcp_kv_gather_kernel<<<grid, 32, kGatherSmem, (cudaStream_t)stream>>>(
        reinterpret_cast<const int4*>(K), reinterpret_cast<const int4*>(V),
        reinterpret_cast<int4*>(k_out) + dst_row * cpr, reinterpret_cast<int4*>(v_out) + dst_row * cpr,
        rg);
    if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
    dst_row += c / cpr;
  }
  return FCP_OK;
}

extern "C" int fcp_kv_scatter_add(const fcp_plan* plan, int32_t rank, const void* dk_r,
                                  const void* dv_r, int32_t src_dtype, float* dK, float* dV,
                                  int32_t n_kv_heads, int32_t head_dim, void* stream,
                                  fcp_gather_counts* counts) {
  return fcp_kv_scatter_add_piece(plan, rank, FCP_PIECE_FULL, dk_r, dv_r, src_dtype, dK, dV,
                                  n_kv_heads, head_dim, stream, counts);
}

extern "C" int fcp_kv_scatter_add_piece(const fcp_plan* plan, int32_t rank, int32_t piece,
                                        const void* dk_r, const void* dv_r, int32_t src_dtype,
                                        float* dK, float* dV, int32_t n_kv_heads, int32_t head_dim,
                                        void* stream, fcp_gather_counts* counts) {
  if (!plan || rank < 0 || rank >= plan->n_ranks || !valid_piece(piece) || !dK || !dV ||
      n_kv_heads < 1 || head_dim < 1)
    return FCP_INVALID_ARG;
  if (src_dtype != FCP_DTYPE_BF16 && src_dtype != FCP_DTYPE_F32) return FCP_UNSUPPORTED;
  const int64_t row_elems = (int64_t)n_kv_heads * head_dim;
  if (row_elems % 8 != 0) return FCP_UNSUPPORTED;
  if (!aligned16(dk_r) || !aligned16(dv_r) || !aligned16(dK) || !aligned16(dV)) return FCP_MISALIGNED;
  RankView v;
  std::vector<int64_t> tok, len;                  // merged destination ranges (global tokens)
  const int st = fcp_guard([&] {
    fcp_build_rank_view(*plan, rank, v, piece);
    for (size_t g = 0; g < v.kv_len.size(); ++g) {
      if (v.kv_len[g] == 0) continue;
      if (!tok.empty() && tok.back() + len.back() == v.kv_src_start[g]) {
        len.back() += v.kv_len[g];
      } else {
        tok.push_back(v.kv_src_start[g]);
        len.push_back(v.kv_len[g]);
      }
    }
    return (int)FCP_OK;
  });
  if (st != FCP_OK) return st;
  if (v.n_kv > 0 && (!dk_r || !dv_r)) return FCP_INVALID_ARG;     // an empty piece needs no buffer
  const int64_t esz = src_dtype == FCP_DTYPE_F32 ? 4 : 2;
  if (counts) {
    counts->total_tokens = v.n_kv;
    counts->remote_tokens = v.remote;
    counts->total_bytes = 2 * v.n_kv * row_elems * esz;      // dk_r and dv_r, one pass
    counts->remote_bytes = 2 * v.remote * row_elems * esz;   // what a ReduceScatter would move
    counts->n_ranges = (int32_t)tok.size();
    counts->reserved = 0;
  }
  const int64_t upr = row_elems / 8;              // 8-element units per row
  const int num_sms = fcp_sm_count();
  int64_t src_row = 0;
  for (size_t base = 0; base < tok.size();) {
    // one launch = a run of buffer-contiguous ranges with pairwise distinct destination tokens.
    // Ranges are in (document, start) order, so a range can only overlap the one before it (a
    // PREFIX piece repeats a prefix when the rank holds two shards of one document): such a
    // range opens the next launch, ordered after this one on the stream.
    GatherRanges rg;
    std::memset(&rg, 0, sizeof(rg));
    int64_t c = 0, run_end = -1;
    while (base < tok.size() && rg.n < kMaxRanges && tok[base] >= run_end) {
      rg.dst0[rg.n] = c;                          // position in the rank buffer
      rg.src0[rg.n] = tok[base] * upr;            // position in the global accumulator
      c += len[base] * upr;
      run_end = std::max(run_end, tok[base] + len[base]);
      ++rg.n;
      ++base;
    }
    rg.dst0[rg.n] = c;
    const int64_t spans = 2 * ((c + kScatterThreads * kScatterUnroll - 1) / (kScatterThreads * kScatterUnroll));
    if (spans == 0) continue;
    const int grid = (int)std::min<int64_t>(spans, (int64_t)num_sms * 8);
    if (src_dtype == FCP_DTYPE_BF16)
      fcp_kv_scatter_add_kernel<__nv_bfloat16><<<grid, kScatterThreads, 0, (cudaStream_t)stream>>>(
          static_cast<const __nv_bfloat16*>(dk_r) + src_row * row_elems,
          static_cast<const __nv_bfloat16*>(dv_r) + src_row * row_elems, dK, dV, rg);
    else
      fcp_kv_scatter_add_kernel<float><<<grid, kScatterThreads, 0, (cudaStream_t)stream>>>(
          static_cast<const float*>(dk_r) + src_row * row_elems,
          static_cast<const float*>(dv_r) + src_row * row_elems, dK, dV, rg);
    if (cudaGetLastError() != cudaSuccess) return FCP_CUDA;
    src_row += c / upr;
  }
  return FCP_OK;
}

extern "C" int fcp_kv_reduce_finish(const float* dK, const float* dV, void* dK_out, void* dV_out,
                                    int64_t n_elems, void* stream) {
  if (n_elems < 0 || n_elems % 8 != 0) return FCP_INVALID_ARG;
  if (n_elems == 0) return FCP_OK;
  if (!dK || !dV || !dK_out || !dV_out) return FCP_INVALID_ARG;
  if (!aligned16(dK) || !aligned16(dV) || !aligned16(dK_out) || !aligned16(dV_out))
    return FCP_MISALIGNED;
  const int64_t n8 = n_elems / 8;
  const int grid = (int)std::min<int64_t>((n8 + 255) / 256, (int64_t)fcp_sm_count() * 8);
  fcp_kv_reduce_finish_kernel<<<dim3(grid, 2), 256, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const float4*>(dK), reinterpret_cast<const float4*>(dV),
      reinterpret_cast<int4*>(dK_out), reinterpret_cast<int4*>(dV_out), n8);
  return cudaGetLastError() == cudaSuccess ? FCP_OK : FCP_CUDA;
}

extern "C" int fcp_merge(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b,
                         void* o_out, float* lse_out, int64_t n_rows, int32_t n_heads,
                         int32_t head_dim, int32_t o_dtype, void* stream) {
  if (n_rows < 0 || n_heads < 1) return FCP_INVALID_ARG;
  if ((head_dim != 64 && head_dim != 128) ||
      (o_dtype != FCP_DTYPE_BF16 && o_dtype != FCP_DTYPE_F32))
    return FCP_UNSUPPORTED;
  if (n_rows == 0) return FCP_OK;                  // empty input: nothing to do, pointers unused
  if (!o_a || !lse_a || !o_b || !lse_b || !o_out || !lse_out) return FCP_INVALID_ARG;
  if (!aligned16(o_a) || !aligned16(o_b) || !aligned16(o_out)) return FCP_MISALIGNED;
  const int64_t threads = n_rows * n_heads * (head_dim / 8);
  const int64_t blocks = (threads + 255) / 256;
  if (blocks > INT32_MAX) return FCP_INVALID_ARG;
  if (o_dtype == FCP_DTYPE_BF16)
    fcp_merge_kernel<__nv_bfloat16><<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(
        o_a, lse_a, o_b, lse_b, o_out, lse_out, n_rows, n_heads, head_dim);
  else
    fcp_merge_kernel<float><<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(
        o_a, lse_a, o_b, lse_b, o_out, lse_out, n_rows, n_heads, head_dim);
  return cudaGetLastError() == cudaSuccess ? FCP_OK : FCP_CUDA;
}

extern "C" int fcp_sched_upload(const fcp_sched* s, void* workspace, void* stream) {
  if (!s || !workspace) return FCP_INVALID_ARG;
  if (!aligned16(workspace)) return FCP_MISALIGNED;
  // The lists were laid out in one host image by fcp_sched_create: a single copy.  The source
  // is pageable host memory owned by the schedule: cudaMemcpyAsync returns once it is staged,
  // so no synchronisation is needed here.
  const bool ok = cudaMemcpyAsync(workspace, s->image.data(), s->image.size(), cudaMemcpyHostToDevice,
                                  (cudaStream_t)stream) == cudaSuccess;
  return ok ? FCP_OK : FCP_CUDA;
}
