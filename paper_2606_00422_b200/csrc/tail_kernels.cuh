// tail_kernels.cuh -- the consumer of the ranking pass: per-action head logits ->
// probabilities -> utility (PAPER.md:146-152, Eq. 4's heads and weights; :321 "head utility
// functions"), and the per-user top-K of the ranked candidates.  Both are
// HBM-bound streaming kernels (no contraction worth a tensor core: the heads' first layers are the
// GEMM, linear_kernel.cuh; what is left is one dot product of length Dh per (candidate, head)).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx.cuh"

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


// Layer normalisation over the hidden dimension of candidate tokens, bf16 in / bf16 out, fp32
// statistics, two passes over registers (D <= 4096, D % 8 == 0): one warp per row, 16-byte loads.  HBM-bound.
constexpr int kLnMaxChunks = 16;   // 16-byte chunks per lane: D <= 32 * 8 * 16 = 4096

// Y_FP8: the output leaves as E4M3 bytes, byte = cvt.rn.satfinite.e4m3(value * y_mult) -- the operand of an FP8
// linear layer (upr_linear_fp8_ex_fwd with x_dtype = UPR_FP8_E4M3), one byte per element instead of two.
template <bool Y_FP8>
__global__ void __launch_bounds__(256) upr_layernorm_kernel(const __nv_bfloat16* __restrict__ x,
                                                            const float* __restrict__ gamma,
                                                            const float* __restrict__ beta, long long M, int D,
                                                            float eps, void* __restrict__ y_out, float y_mult) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = (static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const long long n_warps = (static_cast<long long>(gridDim.x) * blockDim.x) >> 5;
  const int n_chunks = D / 8;   // 16-byte chunks per row
  for (long long m = warp0; m < M; m += n_warps) {
    const uint4* src = reinterpret_cast<const uint4*>(x + m * D);
    float v[kLnMaxChunks][8];
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < kLnMaxChunks; ++i) {
      const int c = i * 32 + lane;
      if (c < n_chunks) {
        const uint4 q = __ldg(src + c);
        const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          v[i][2 * k] = __uint_as_float(w[k] << 16);
          v[i][2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
          sum += v[i][2 * k] + v[i][2 * k + 1];
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    const float mean = sum / static_cast<float>(D);
    float sq = 0.f;
#pragma unroll
    for (int i = 0; i < kLnMaxChunks; ++i)
      if (i * 32 + lane < n_chunks) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const float c = v[i][k] - mean;
          sq = fmaf(c, c, sq);
        }
      }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
    const float rstd = rsqrtf(sq / static_cast<float>(D) + eps);
    uint4* dst = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(y_out) + m * D);
    uint2* dst8 = reinterpret_cast<uint2*>(static_cast<uint8_t*>(y_out) + m * D);
#pragma unroll
    for (int i = 0; i < kLnMaxChunks; ++i) {
      const int c = i * 32 + lane;
      if (c < n_chunks) {
        const float4 g0 = __ldg(reinterpret_cast<const float4*>(gamma + c * 8));
        const float4 g1 = __ldg(reinterpret_cast<const float4*>(gamma + c * 8 + 4));
        const float4 b0 = __ldg(reinterpret_cast<const float4*>(beta + c * 8));
        const float4 b1 = __ldg(reinterpret_cast<const float4*>(beta + c * 8 + 4));
        const float g[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
        const float b[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
        uint32_t o[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float lo = fmaf((v[i][2 * k] - mean) * rstd, g[2 * k], b[2 * k]);
          const float hi = fmaf((v[i][2 * k + 1] - mean) * rstd, g[2 * k + 1], b[2 * k + 1]);
          if (Y_FP8)
            o[k] = __nv_cvt_float2_to_fp8x2(make_float2(lo * y_mult, hi * y_mult), __NV_SATFINITE, __NV_E4M3);
          else
            o[k] = pack_bf16x2(lo, hi);
        }
        if (Y_FP8) dst8[c] = make_uint2(o[0] | (o[1] << 16), o[2] | (o[3] << 16));
        else dst[c] = make_uint4(o[0], o[1], o[2], o[3]);
      }
    }
  }
}

}  // namespace upr
