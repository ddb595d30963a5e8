// pack_kernels.cuh -- step a1: pool slot -> packed decode cache (pool shape
// [layers, slots, heads, n, D] PAPER.md:202), optional FP8 E4M3 quantisation with
// per-(layer, head) scales; and step a8: split-K combine.  All HBM-bound: 16-byte vector
// accesses, one warp per 16-row block (a block never straddles two users because user blocks
// start on multiples of 16 rows), persistent grid-stride loops sized to the SM count.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace upr {

constexpr int kPackThreads = 256;
constexpr int kPackRowBlock = 16;  // == UPR_ROW_ALIGN

// Build row_off[0..B] (aligned exclusive prefix of seq_lens) in shared memory.
__device__ __forceinline__ void build_row_off(const int32_t* __restrict__ seq_lens, int B,
                                              int* row_off /* smem [B+1] */) {
  // serial-by-chunks scan: thread 0 of the CTA is enough for B up to a few thousand, but do it
  // with the whole CTA: each thread sums a contiguous chunk, then a scan over chunk sums.
  __shared__ int chunk_sum[kPackThreads];
  const int tid = threadIdx.x;
  const int per = (B + kPackThreads - 1) / kPackThreads;
  const int lo = min(B, tid * per), hi = min(B, lo + per);
  int s = 0;
  for (int b = lo; b < hi; ++b) s += (__ldg(seq_lens + b) + kPackRowBlock - 1) / kPackRowBlock * kPackRowBlock;
  chunk_sum[tid] = s;
  __syncthreads();
  if (tid == 0) {
    int acc = 0;
    for (int i = 0; i < kPackThreads; ++i) {
      int v = chunk_sum[i];
      chunk_sum[i] = acc;
      acc += v;
    }
    row_off[B] = acc;
  }
  __syncthreads();
  int acc = chunk_sum[tid];
  for (int b = lo; b < hi; ++b) {
    row_off[b] = acc;
    acc += (__ldg(seq_lens + b) + kPackRowBlock - 1) / kPackRowBlock * kPackRowBlock;
  }
  __syncthreads();
}

// largest b with row_off[b] <= row  (row < row_off[B]); users with zero rows are skipped
__device__ __forceinline__ int find_user(const int* row_off, int B, int row) {
  int lo = 0, hi = B;  // invariant: row_off[lo] <= row < row_off[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (row_off[mid] <= row) lo = mid; else hi = mid;
  }
  return lo;
}

struct PackArgs {
  const __nv_bfloat16* pool;  // [n_layers, S, H, n_max, d]
  void* cache;                // packed [n_layers, H, R, d] + tail
  float* scale;               // FP8: holds amax while packing, scale after finalize
  const int32_t* slot_ids;
  const int32_t* seq_lens;
  int B, H, d, n_layers, S, n_max, tail_rows;
  int per_user;               // FP8: one scale per (layer, user, head) instead of per (layer, head)
};

// MODE 0: bf16 copy, 1: fp8 quantise, 2: fp32 widen, 3: amax pass (no cache write)
// Each warp owns a CONTIGUOUS range of 16-row blocks (it streams a contiguous piece of the
// cache; the amax pass then needs one atomic per (layer, head) change instead of one per
// block) and keeps U blocks' worth of 16-byte loads in flight before it converts and stores.
template <int MODE, int D>
__global__ void __launch_bounds__(kPackThreads) upr_pack_kernel(const PackArgs a) {
  extern __shared__ int row_off[];  // [B+1]
  build_row_off(a.seq_lens, a.B, row_off);
  const int R = row_off[a.B];
  const int blocks_per_head = R / kPackRowBlock;
  const long long n_blocks = static_cast<long long>(a.n_layers) * a.H * blocks_per_head;
  const int lane = threadIdx.x & 31;
  constexpr int kWarpsPerCta = kPackThreads / 32;
  const long long n_warps = static_cast<long long>(gridDim.x) * kWarpsPerCta;
  const long long wid = static_cast<long long>(blockIdx.x) * kWarpsPerCta + (threadIdx.x >> 5);
  const long long per = (n_blocks + n_warps - 1) / n_warps;
  const long long blk0 = wid * per;
  const long long blk1 = (blk0 + per < n_blocks) ? (blk0 + per) : n_blocks;
  constexpr int CPR = D / 8;                       // 16-byte bf16 chunks per row
  constexpr int CH = kPackRowBlock * CPR;          // chunks per 16-row block: 128 (d=64) / 256
  constexpr int NI = CH / 32;                      // chunks per lane per block
  constexpr int U = (D == 64) ? 4 : 2;             // blocks in flight per warp

  int cur_lh = -1;        // amax pass: (layer, head) of the running maximum
  float run_max = 0.f;
  // The warp walks its blocks in order, so (layer * H + head, row block, user) are carried along instead of being
  // recomputed per block (a 64-bit division, a modulo and a binary search over the users cost more than moving the
  // block's 2 - 4 KB: the d = 64 passes ran at 4.3 - 4.8 TB/s with the ALU pipe at 35 - 43 %).
  int w_lh = 0, w_rb = 0, w_b = 0;
  if (blk0 < blk1) {
    w_lh = static_cast<int>(blk0 / blocks_per_head);
    w_rb = static_cast<int>(blk0 - static_cast<long long>(w_lh) * blocks_per_head);
    w_b = find_user(row_off, a.B, w_rb * kPackRowBlock);
  }
  int w_l = w_lh / a.H, w_h = w_lh - w_l * a.H;
  for (long long blk = blk0; blk < blk1; blk += U) {
    uint4 v[U][NI];
    size_t dst_elem[U];
    int lh_u[U];
    float mult[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const long long bk = blk + u;
      lh_u[u] = -1;
      dst_elem[u] = 0;
      mult[u] = 1.0f;
#pragma unroll
      for (int i = 0; i < NI; ++i) v[u][i] = make_uint4(0u, 0u, 0u, 0u);
      if (bk < blk1) {
        const int lh = w_lh, h = w_h, l = w_l;
        const int row = w_rb * kPackRowBlock;
        while (row >= row_off[w_b + 1]) ++w_b;               // (users without rows are skipped)
        const int b = w_b;
        if (++w_rb == blocks_per_head) {                     // next block: first rows of the next (layer, head)
          w_rb = 0;
          w_b = 0;
          ++w_lh;
          if (++w_h == a.H) {
            w_h = 0;
            ++w_l;
          }
        }
        const int j0 = row - row_off[b];                     // first key index of this block
        const int valid_rows = max(0, min(kPackRowBlock, __ldg(a.seq_lens + b) - j0));
        const int slot = __ldg(a.slot_ids + b);
        const __nv_bfloat16* src =
            a.pool + ((((static_cast<size_t>(l) * a.S + slot) * a.H + h) * a.n_max) + j0) * D;
        // index of the scale (and, in the amax pass, of the running maximum) this block belongs to
        lh_u[u] = a.per_user ? (l * a.B + b) * a.H + h : lh;
        dst_elem[u] = (static_cast<size_t>(lh) * R + row) * D;
        const int valid_chunks = valid_rows * CPR;
        if (MODE == 1) {
          const float amax = a.scale[lh_u[u]];
          mult[u] = amax > 0.f ? __fdiv_rn(448.0f, amax) : 1.0f;
        }
#pragma unroll
        for (int i = 0; i < NI; ++i) {
          const int c = i * 32 + lane;
          if (c < valid_chunks) v[u][i] = __ldg(reinterpret_cast<const uint4*>(src) + c);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (lh_u[u] < 0) continue;
      if constexpr (MODE == 3) {
        // the maximum of bf16 magnitudes is exact in bf16: packed HMNMX2 on the raw pairs, widened once per block
        __nv_bfloat162 m2a = __float2bfloat162_rn(0.f), m2b = m2a;
#pragma unroll
        for (int i = 0; i < NI; ++i) {
          const __nv_bfloat162* p2 = reinterpret_cast<const __nv_bfloat162*>(&v[u][i]);
          m2a = __hmax2(m2a, __hmax2(__habs2(p2[0]), __habs2(p2[1])));
          m2b = __hmax2(m2b, __hmax2(__habs2(p2[2]), __habs2(p2[3])));
        }
        const float2 mf = __bfloat1622float2(__hmax2(m2a, m2b));
        const float wmax = fmaxf(mf.x, mf.y);
        if (lh_u[u] != cur_lh) {
          // flush the finished (layer, head): non-negative floats order like their bit patterns
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) run_max = fmaxf(run_max, __shfl_xor_sync(0xffffffffu, run_max, o));
          if (lane == 0 && cur_lh >= 0 && run_max > 0.f)
            atomicMax(reinterpret_cast<unsigned int*>(a.scale + cur_lh), __float_as_uint(run_max));
          cur_lh = lh_u[u];
          run_max = 0.f;
        }
        run_max = fmaxf(run_max, wmax);
      } else {
#pragma unroll
      for (int i = 0; i < NI; ++i) {
        const int c = i * 32 + lane;
        const uint4 x = v[u][i];
        const __nv_bfloat162* p2 = reinterpret_cast<const __nv_bfloat162*>(&x);
        if (MODE == 0) {
          reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(a.cache) + dst_elem[u])[c] = x;
        } else if (MODE == 1) {
          uint32_t w[2];
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const float2 f0 = __bfloat1622float2(p2[2 * k]), f1 = __bfloat1622float2(p2[2 * k + 1]);
            const uint16_t lo16 = __nv_cvt_float2_to_fp8x2(
                make_float2(__fmul_rn(f0.x, mult[u]), __fmul_rn(f0.y, mult[u])), __NV_SATFINITE, __NV_E4M3);
            const uint16_t hi16 = __nv_cvt_float2_to_fp8x2(
                make_float2(__fmul_rn(f1.x, mult[u]), __fmul_rn(f1.y, mult[u])), __NV_SATFINITE, __NV_E4M3);
            w[k] = static_cast<uint32_t>(lo16) | (static_cast<uint32_t>(hi16) << 16);
          }
          reinterpret_cast<uint2*>(static_cast<uint8_t*>(a.cache) + dst_elem[u])[c] = make_uint2(w[0], w[1]);
        } else {
          float4 o0, o1;
          float2 f;
          f = __bfloat1622float2(p2[0]); o0.x = f.x; o0.y = f.y;
          f = __bfloat1622float2(p2[1]); o0.z = f.x; o0.w = f.y;
          f = __bfloat1622float2(p2[2]); o1.x = f.x; o1.y = f.y;
          f = __bfloat1622float2(p2[3]); o1.z = f.x; o1.w = f.y;
          float4* dp = reinterpret_cast<float4*>(static_cast<float*>(a.cache) + dst_elem[u]) + 2 * c;
          dp[0] = o0;
          dp[1] = o1;
        }
      }
      }
    }
  }
  if (MODE == 3) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) run_max = fmaxf(run_max, __shfl_xor_sync(0xffffffffu, run_max, o));
    if (lane == 0 && cur_lh >= 0 && run_max > 0.f)
      atomicMax(reinterpret_cast<unsigned int*>(a.scale + cur_lh), __float_as_uint(run_max));
  }
  if (MODE != 3) {
    // zero the tail rows after the last (layer, head) block
    const size_t tail0 = static_cast<size_t>(a.n_layers) * a.H * R * D;  // element index
    const size_t eb = (MODE == 0) ? 2 : (MODE == 1) ? 1 : 4;
    const size_t n16 = static_cast<size_t>(a.tail_rows) * D * eb / 16;
    uint4* tp = reinterpret_cast<uint4*>(static_cast<uint8_t*>(a.cache) + tail0 * eb);
    for (size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n16;
         i += static_cast<size_t>(gridDim.x) * blockDim.x)
      tp[i] = make_uint4(0u, 0u, 0u, 0u);
  }
}

// amax -> scale = amax / 448 (amax == 0 -> 1), in place
__global__ void upr_scale_finalize_kernel(float* scale, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    float amax = scale[i];
    scale[i] = amax > 0.f ? __fdiv_rn(amax, 448.0f) : 1.0f;
  }
}

// ---------------------------------------------------------------------------------------
// a8: combine split-K partial states.  part_o [rows][ns][D], part_ml [rows][ns][2] with
// rows = n_layers*total_q*H; m in log2 units.  One warp per output row.
//   m* = max_i m_i; out = sum_i O~_i 2^(m_i - m*) / sum_i l_i 2^(m_i - m*); all empty -> 0.
// ---------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(256) upr_combine_kernel(const float* __restrict__ part_o,
                                                          const float* __restrict__ part_ml,
                                                          float* __restrict__ out, long long rows,
                                                          int ns) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = static_cast<long long>(blockIdx.x) * 8 + (threadIdx.x >> 5);
  const long long stride = static_cast<long long>(gridDim.x) * 8;
  constexpr int V = D / 32;  // floats per lane
  for (long long r = warp0; r < rows; r += stride) {
    const float* ml = part_ml + r * ns * 2;
    float mstar = -INFINITY;
    for (int i = 0; i < ns; ++i) mstar = fmaxf(mstar, __ldg(ml + 2 * i));
    float acc[V];
#pragma unroll
    for (int k = 0; k < V; ++k) acc[k] = 0.f;
    float lstar = 0.f;
    if (mstar > -INFINITY) {
      for (int i = 0; i < ns; ++i) {
        const float mi = __ldg(ml + 2 * i);
        if (mi == -INFINITY) continue;
        const float f = exp2f(mi - mstar);
        lstar = fmaf(__ldg(ml + 2 * i + 1), f, lstar);
        const float* po = part_o + (r * ns + i) * D + lane * V;
        if (V == 2) {
          float2 v = __ldg(reinterpret_cast<const float2*>(po));
          acc[0] = fmaf(v.x, f, acc[0]);
          acc[1] = fmaf(v.y, f, acc[1]);
        } else {
          float4 v = __ldg(reinterpret_cast<const float4*>(po));
          acc[0] = fmaf(v.x, f, acc[0]);
          acc[1] = fmaf(v.y, f, acc[1]);
          acc[2] = fmaf(v.z, f, acc[2]);
          acc[3] = fmaf(v.w, f, acc[3]);
        }
      }
    }
    const float inv = lstar > 0.f ? 1.0f / lstar : 0.f;
    float* po = out + r * D + lane * V;
    if (V == 2) {
      *reinterpret_cast<float2*>(po) = make_float2(acc[0] * inv, acc[1] * inv);
    } else {
      *reinterpret_cast<float4*>(po) = make_float4(acc[0] * inv, acc[1] * inv, acc[2] * inv, acc[3] * inv);
    }
  }
}

}  // namespace upr
