// linear_kernel.cuh -- y = act(x W^T + b) over candidate tokens: the linear layers around the
// ranking cross-attention (out-projection, MLP, Q / self-K,V projections, the stacked first layers of
// the per-action heads, "only the candidate tokens are processed").
//
// A dense contraction, so it runs on the tensor cores: persistent, warp-specialised tcgen05 GEMM,
// 128 x 128 output tiles, K in steps of 64 (one 128-byte swizzled row per operand row):
//   warp 0      TMA producer: x tile [128 rows, 64 k] and W tile [128 outputs, 64 k] per stage
//   warp 1      tcgen05.mma issuer (one elected thread), fp32 accumulators in TMEM, two of them so
//               that the epilogue of tile i overlaps the MMAs of tile i + 1
//   warps 2-3, 8-9  converters (fp32 x only, e.g. the attention output): raw fp32 rows -> bf16 swizzled
//               MMA tile, so the activation never takes a separate cast pass through HBM
//   warps 4-7   epilogue: TMEM -> registers, + bias, activation, store as bf16 or fp32
// x: [M, K] bf16 or fp32 row-major; W: [N, K] bf16 row-major (one output feature per row);
// y: [M, N] bf16 or fp32 row-major.  K % 64 == 0, N % 8 == 0; M is arbitrary (TMA clips the
// last tile's rows and zero-fills, stores are predicated).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <cuda/std/type_traits>

#include "ptx.cuh"

namespace upr {
namespace lin {

constexpr int kThreads = 320;
constexpr int kBM = 128, kBN = 128, kBK = 64;
constexpr int kTileBytes = kBM * kBK * 2;      // 16 KB: one bf16 operand tile
constexpr int kRawBytes = kBM * kBK * 4;       // 32 KB: one fp32 x tile as loaded
constexpr int kStages = 5;                     // (x, W) tile pairs
constexpr int kRawStages = 2;
constexpr int kConvThreads = 128;          // warps 2, 3, 8, 9
constexpr int kSmemCtrl = 1024;
constexpr int kSmemTotal = kStages * 2 * kTileBytes + kRawStages * kRawBytes + kSmemCtrl + 1024;
static_assert(kSmemTotal <= 232448, "exceeds the 227 KB shared memory of an sm_100 CTA");

enum : int { ACT_NONE = 0, ACT_SILU = 1, ACT_RELU = 2 };

struct Args {
  const float* bias;      // [N] fp32 or nullptr
  const __nv_bfloat16* residual;   // [M, N] bf16 added after the activation (the residual stream), or nullptr
  void* y;                // [M, N] bf16 or fp32
  long long M;
  int N, K;
  int act;
  int y_is_f32;
  float out_scale;        // multiplies the accumulator before the bias (FP8 operands: x_scale * w_scale; else 1)
  float x_mult;           // FP8 operands: x is quantised as e4m3(x * x_mult), x_mult = 1 / x_scale
  int y_is_fp8;           // pair kernel only: y is e4m3 [M, N], byte = cvt.rn.satfinite.e4m3(value * y_mult)
  float y_mult;           // 1 / y_scale
  // K/V projection written straight into the pool layout [layers, S, H, n, d]: row m of y is token
  // m's [H, d] vector and goes to pool[layer, tok_slot[m], h, tok_pos[m], :]; y = the pool (bf16), N = H * d
  const int32_t* tok_slot;
  const int32_t* tok_pos;
  int kv_layer, kv_S, kv_H, kv_n, kv_d;
};

struct __align__(16) Ctrl {
  uint64_t full[kStages], empty[kStages];
  uint64_t raw_full[kRawStages], raw_empty[kRawStages];
  uint64_t acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= kSmemCtrl, "control block too large");

template <bool X_F32>
__global__ void __launch_bounds__(kThreads, 1)
upr_linear_kernel(const __grid_constant__ CUtensorMap tmap_x,   // bf16: box 128 x 64, SWIZZLE_128B; fp32: box 128 x 64, no swizzle
                  const __grid_constant__ CUtensorMap tmap_w,   // bf16 [N, K], box 128 x 64, SWIZZLE_128B
                  const Args args) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_aligned = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t a_smem = smem_base;                               // kStages x tiles
  const uint32_t b_smem = a_smem + kStages * kTileBytes;           // kStages W tiles
  const uint32_t raw_smem = b_smem + kStages * kTileBytes;         // kRawStages fp32 x tiles
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_aligned + kStages * 2 * kTileBytes + kRawStages * kRawBytes);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m_tiles = static_cast<int>((args.M + kBM - 1) / kBM);
  const int n_tiles = (args.N + kBN - 1) / kBN;
  const int k_steps = args.K / kBK;
  const long long total_tiles = static_cast<long long>(m_tiles) * n_tiles;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) {
      // fp32 x: the W bytes (producer's arrive.expect_tx) and the four converter warps complete a stage
      mbar_init(smem_u32(&ctrl->full[i]), X_F32 ? 5 : 1);
      mbar_init(smem_u32(&ctrl->empty[i]), 1);
    }
    for (int i = 0; i < kRawStages; ++i) {
      mbar_init(smem_u32(&ctrl->raw_full[i]), 1);
      mbar_init(smem_u32(&ctrl->raw_empty[i]), 4);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl->acc_full[i]), 1);
      mbar_init(smem_u32(&ctrl->acc_empty[i]), 4);
    }
    fence_mbar_init();
  }
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmap_x);
    tma_prefetch_desc(&tmap_w);
  }
  if (warp == 1) {
    tmem_alloc(smem_u32(&ctrl->tmem_base), 256);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;

  if (warp == 0) {
    // ================================================================= producer
    if (elect_one()) {
      uint32_t it = 0, raw_it = 0;
      for (long long t = blockIdx.x; t < total_tiles; t += gridDim.x) {
        const int mb = static_cast<int>(t / n_tiles), nb = static_cast<int>(t % n_tiles);
        for (int ks = 0; ks < k_steps; ++ks, ++it) {
          const uint32_t s = it % kStages, ph = (it / kStages) & 1;
          mbar_wait<1>(smem_u32(&ctrl->empty[s]), ph ^ 1);
          const uint32_t full = smem_u32(&ctrl->full[s]);
          if (X_F32) {
            mbar_arrive_expect_tx(full, kTileBytes);
            tma_load_2d(b_smem + s * kTileBytes, &tmap_w, ks * kBK, nb * kBN, full);
            const uint32_t rs = raw_it % kRawStages, rph = (raw_it / kRawStages) & 1;
            mbar_wait<2>(smem_u32(&ctrl->raw_empty[rs]), rph ^ 1);
            const uint32_t rfull = smem_u32(&ctrl->raw_full[rs]);
            mbar_arrive_expect_tx(rfull, kRawBytes);
            tma_load_2d(raw_smem + rs * kRawBytes, &tmap_x, ks * kBK, mb * kBM, rfull);
            ++raw_it;
          } else {
            mbar_arrive_expect_tx(full, 2 * kTileBytes);
            tma_load_2d(a_smem + s * kTileBytes, &tmap_x, ks * kBK, mb * kBM, full);
            tma_load_2d(b_smem + s * kTileBytes, &tmap_w, ks * kBK, nb * kBN, full);
          }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================================================================= MMA issuer
    if (elect_one()) {
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO 1024, version 1, SWIZZLE_128B
      constexpr uint32_t kLoK = (16u >> 4) << 16;
      constexpr uint32_t kIdesc = make_idesc_bf16(kBM, kBN, 0, 0);
      auto mk_desc = [](uint32_t lo) {
        return (static_cast<uint64_t>(kDescHi) << 32) | static_cast<uint64_t>(lo);
      };
      const uint32_t a_lo = ((a_smem & 0x3FFFFu) >> 4) | kLoK;
      const uint32_t b_lo = ((b_smem & 0x3FFFFu) >> 4) | kLoK;
      uint32_t it = 0, n_acc = 0;
      for (long long t = blockIdx.x; t < total_tiles; t += gridDim.x, ++n_acc) {
        const uint32_t ab = n_acc & 1;
        if (n_acc >= 2) mbar_wait<3>(smem_u32(&ctrl->acc_empty[ab]), ((n_acc >> 1) - 1) & 1);
        tc_fence_after();
        for (int ks = 0; ks < k_steps; ++ks, ++it) {
          const uint32_t s = it % kStages, ph = (it / kStages) & 1;
          mbar_wait<4>(smem_u32(&ctrl->full[s]), ph);
          tc_fence_after();
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k)
            umma_ss(tmem_base + ab * kBN, mk_desc(a_lo + ((s * kTileBytes + k * 32) >> 4)),
                    mk_desc(b_lo + ((s * kTileBytes + k * 32) >> 4)), kIdesc, (ks > 0 || k > 0) ? 1u : 0u);
          umma_commit(smem_u32(&ctrl->empty[s]));
        }
        umma_commit(smem_u32(&ctrl->acc_full[ab]));
      }
    }
    __syncwarp();
  } else if (warp == 2 || warp == 3 || warp >= 8) {
    // ================================================================= converters (fp32 x)
    if constexpr (X_F32) {
      const int ctid = (warp < 4 ? warp - 2 : warp - 6) * 32 + lane;   // 0..127
      uint32_t it = 0, raw_it = 0;
      for (long long t = blockIdx.x; t < total_tiles; t += gridDim.x) {
        for (int ks = 0; ks < k_steps; ++ks, ++it, ++raw_it) {
          const uint32_t s = it % kStages, ph = (it / kStages) & 1;
          const uint32_t rs = raw_it % kRawStages, rph = (raw_it / kRawStages) & 1;
          mbar_wait<5>(smem_u32(&ctrl->empty[s]), ph ^ 1);      // the MMA has finished with this stage's x tile
          mbar_wait<6>(smem_u32(&ctrl->raw_full[rs]), rph);
          const uint32_t raw = raw_smem + rs * kRawBytes;
          const uint32_t tile = a_smem + s * kTileBytes;
#pragma unroll 4
          for (int p = ctid; p < kBM * 8; p += kConvThreads) {
            const int row = p >> 3, c8 = p & 7;                  // 8 floats -> one 16-byte bf16 chunk
            const uint4 a = lds128(raw + row * 256 + c8 * 32), b = lds128(raw + row * 256 + c8 * 32 + 16);
            sts128(tile + row * 128 + ((c8 ^ (row & 7)) << 4),
                   pack_bf16x2(__uint_as_float(a.x), __uint_as_float(a.y)),
                   pack_bf16x2(__uint_as_float(a.z), __uint_as_float(a.w)),
                   pack_bf16x2(__uint_as_float(b.x), __uint_as_float(b.y)),
                   pack_bf16x2(__uint_as_float(b.z), __uint_as_float(b.w)));
          }
          fence_proxy_async_smem();   // generic-proxy tile writes -> visible to tcgen05.mma
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(smem_u32(&ctrl->raw_empty[rs]));
            mbar_arrive(smem_u32(&ctrl->full[s]));
          }
        }
      }
    }
  } else {
    // ================================================================= epilogue (warps 4-7)
    const int ew = warp - 4;                                   // TMEM lane quarter
    const uint32_t lane_base = static_cast<uint32_t>(ew * 32) << 16;
    uint32_t n_acc = 0;
    for (long long t = blockIdx.x; t < total_tiles; t += gridDim.x, ++n_acc) {
      const int mb = static_cast<int>(t / n_tiles), nb = static_cast<int>(t % n_tiles);
      const uint32_t ab = n_acc & 1;
      mbar_wait<7>(smem_u32(&ctrl->acc_full[ab]), (n_acc >> 1) & 1);
      tc_fence_after();
      const long long row = static_cast<long long>(mb) * kBM + ew * 32 + lane;
      const bool row_ok = row < args.M;
      // pool mode: first pool row of this token's slot (head 0), or -1
      long long kv_row0 = -1;
      if (args.tok_slot != nullptr && row_ok)
        kv_row0 = ((static_cast<long long>(args.kv_layer) * args.kv_S + __ldg(args.tok_slot + row)) * args.kv_H) * args.kv_n +
                  __ldg(args.tok_pos + row);
      // one 32-column chunk: + bias, activation, store.  The activation is a compile-time branch (the
      // per-element form with run-time tests made the epilogue, not the MMAs, the bound of the kernel)
      auto chunk = [&](auto act_tag, const int c0) {
        constexpr int kAct = decltype(act_tag)::value;
        uint32_t r[32];
        tmem_ld32(tmem_base + lane_base + ab * kBN + c0, r);
        tmem_wait_ld_regs(r);
        if (c0 + 32 == kBN) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl->acc_empty[ab]));
        }
        const int col0 = nb * kBN + c0;
        if (col0 >= args.N || !row_ok) return;
        // N % 8 == 0: 8-column groups are either whole or absent
#pragma unroll
        for (int c = 0; c < 32; c += 8) {
          if (col0 + c >= args.N) break;
          float v[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) v[k] = __uint_as_float(r[c + k]);
          if (args.bias != nullptr) {
            const float4 b0 = __ldg(reinterpret_cast<const float4*>(args.bias + col0 + c));
            const float4 b1 = __ldg(reinterpret_cast<const float4*>(args.bias + col0 + c + 4));
            v[0] += b0.x; v[1] += b0.y; v[2] += b0.z; v[3] += b0.w;
            v[4] += b1.x; v[5] += b1.y; v[6] += b1.z; v[7] += b1.w;
          }
          if (kAct == ACT_SILU) {
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = __fdividef(v[k], 1.0f + __expf(-v[k]));
          } else if (kAct == ACT_RELU) {
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = fmaxf(v[k], 0.f);
          }
          if (args.residual != nullptr) {
            const uint4 q = __ldg(reinterpret_cast<const uint4*>(args.residual + row * args.N + col0 + c));
            const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              v[2 * k] += __uint_as_float(w[k] << 16);
              v[2 * k + 1] += __uint_as_float(w[k] & 0xffff0000u);
            }
          }
          if (args.tok_slot != nullptr) {
            const int col = col0 + c, h = col / args.kv_d, t = col - h * args.kv_d;   // 8 columns stay inside one head
            __nv_bfloat16* dst = static_cast<__nv_bfloat16*>(args.y) +
                                 (kv_row0 + static_cast<long long>(h) * args.kv_n) * args.kv_d + t;
            *reinterpret_cast<uint4*>(dst) = make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]),
                                                        pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
          } else if (args.y_is_f32) {
            float* dst = static_cast<float*>(args.y) + row * args.N + col0 + c;
            *reinterpret_cast<float4*>(dst) = make_float4(v[0], v[1], v[2], v[3]);
            *reinterpret_cast<float4*>(dst + 4) = make_float4(v[4], v[5], v[6], v[7]);
          } else {
            __nv_bfloat16* dst = static_cast<__nv_bfloat16*>(args.y) + row * args.N + col0 + c;
            *reinterpret_cast<uint4*>(dst) = make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]),
                                                        pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
          }
        }
      };
#pragma unroll 1
      for (int c0 = 0; c0 < kBN; c0 += 32) {
        if (args.act == ACT_SILU) chunk(cuda::std::integral_constant<int, ACT_SILU>{}, c0);
        else if (args.act == ACT_RELU) chunk(cuda::std::integral_constant<int, ACT_RELU>{}, c0);
        else chunk(cuda::std::integral_constant<int, ACT_NONE>{}, c0);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 256);
  }
}

}  // namespace lin
}  // namespace upr
