// tail_kernels.cuh -- the consumer of the ranking pass: per-action head logits ->
// probabilities -> utility (PAPER.md:146-152, Eq. 4's heads and weights; :321 "head utility
// functions"), and the per-user top-K of the ranked candidates.  Both are
// HBM-bound streaming kernels (no contraction worth a tensor core: the heads' first layers are the
// GEMM, linear_kernel.cuh; what is left is one dot product of length Dh per (candidate, head)).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace upr {

// hid [M, C*Dh] bf16 = act(W1_c z + b1_c) for the C heads side by side; w2 [C, Dh], b2 [C], wc [C] fp32.
// One warp per candidate row: logit_c = <w2_c, hid_c> + b2_c, p_c = sigmoid(logit_c), u = sum_c wc_c p_c.
__global__ void __launch_bounds__(256) upr_head_utility_kernel(const __nv_bfloat16* __restrict__ hid,
                                                               const float* __restrict__ w2,
                                                               const float* __restrict__ b2,
                                                               const float* __restrict__ wc, long long M, int C,
                                                               int Dh, float* __restrict__ probs,
                                                               float* __restrict__ util) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = (static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const long long n_warps = (static_cast<long long>(gridDim.x) * blockDim.x) >> 5;
  for (long long m = warp0; m < M; m += n_warps) {
    const __nv_bfloat16* row = hid + m * C * Dh;
    float u = 0.f;
    for (int c = 0; c < C; ++c) {
      float acc = 0.f;
      // Dh % 8 == 0: 16-byte loads, 8 elements per lane and step
      for (int j = lane * 8; j < Dh; j += 256) {
        const uint4 x = __ldg(reinterpret_cast<const uint4*>(row + c * Dh + j));
        const float4 wa = __ldg(reinterpret_cast<const float4*>(w2 + c * Dh + j));
        const float4 wb = __ldg(reinterpret_cast<const float4*>(w2 + c * Dh + j + 4));
        const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
        const float ws[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          acc = fmaf(__uint_as_float(xs[k] << 16), ws[2 * k], acc);
          acc = fmaf(__uint_as_float(xs[k] & 0xffff0000u), ws[2 * k + 1], acc);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      const float p = 1.0f / (1.0f + __expf(-(acc + __ldg(b2 + c))));
      if (probs != nullptr && lane == 0) probs[m * C + c] = p;
      u = fmaf(__ldg(wc + c), p, u);
    }
    if (lane == 0) util[m] = u;
  }
}

// Per-user top-K by utility, descending; equal utilities by ascending candidate index (so the
// result is unique).  One CTA per user: 64-bit keys (order-reversed utility bits, local index) in
// shared memory, bitonic sort ascending, first K written out.  out_idx [B, K] holds GLOBAL candidate
// indices, -1 past the user's count.
constexpr int kTopkThreads = 512;

__global__ void __launch_bounds__(kTopkThreads) upr_topk_kernel(const float* __restrict__ util,
                                                                const int32_t* __restrict__ cand_offsets, int K,
                                                                int n_pad,   // power of two >= max candidates per user
                                                                int32_t* __restrict__ out_idx,
                                                                int32_t* __restrict__ out_cnt) {
  extern __shared__ unsigned long long keys[];
  const int b = blockIdx.x;
  const int c0 = __ldg(cand_offsets + b), n = __ldg(cand_offsets + b + 1) - c0;
  for (int i = threadIdx.x; i < n_pad; i += kTopkThreads) {
    unsigned long long key = ~0ull;
    if (i < n) {
      uint32_t bits = __float_as_uint(__ldg(util + c0 + i));
      if (bits == 0x80000000u) bits = 0u;                                  // -0 == +0
      const uint32_t asc = (bits & 0x80000000u) ? ~bits : (bits | 0x80000000u);   // ascending in the float order
      key = (static_cast<unsigned long long>(~asc) << 32) | static_cast<unsigned int>(i);
    }
    keys[i] = key;
  }
  __syncthreads();
  for (int k = 2; k <= n_pad; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < n_pad; i += kTopkThreads) {
        const int ixj = i ^ j;
        if (ixj > i) {
          const unsigned long long x = keys[i], y = keys[ixj];
          if ((x > y) == ((i & k) == 0)) {
            keys[i] = y;
            keys[ixj] = x;
          }
        }
      }
      __syncthreads();
    }
  }
  const int kk = n < K ? n : K;
  for (int r = threadIdx.x; r < K; r += kTopkThreads)
    out_idx[static_cast<long long>(b) * K + r] = r < kk ? c0 + static_cast<int>(keys[r] & 0xffffffffu) : -1;
  if (threadIdx.x == 0) out_cnt[b] = kk;
}

}  // namespace upr
