// linear2_kernel.cuh -- y = act(x W^T + b) [+ residual] on a CTA PAIR: the same layer as linear_kernel.cuh
// (same Args, same epilogue options) with 256 x 256 output tiles over two SMs.
//
// tcgen05.mma.cta_group::2, M = 256 (each CTA holds 128 rows of x and of the accumulator), N = 256 (each CTA
// streams HALF of the W tile: 128 output features x 64 k): an operand byte now feeds 64 MACs instead of 32, i.e.
// half the L2 -> shared-memory traffic per FLOP of the 128 x 128 single-CTA kernel, which is what bounded it.
// Per CTA and k-step: 16 KB of x + 16 KB of W for 512 cycles of MMA.  TMEM: two accumulators of 256 columns
// (the epilogue of tile i overlaps the MMAs of tile i + 1).  Loads of both CTAs complete on the leader's
// barrier, commits are multicast to both CTAs, the peer's epilogue / converter warps arrive remotely.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <cuda/std/type_traits>

#include "linear_kernel.cuh"
#include "ptx.cuh"

namespace upr {
namespace lin2 {

using lin::Args;
using lin::ACT_NONE;
using lin::ACT_RELU;
using lin::ACT_SILU;

constexpr int kThreads = 448;                   // warps: 0 producer, 1 MMA, 2-3 + 8-9 converters, 4-7 + 10-13 epilogue
constexpr int kBM = 256, kBN = 256, kBK = 64;   // per pair; each CTA: 128 rows of x, 128 rows of W
constexpr int kTileBytes = 128 * kBK * 2;       // 16 KB: one CTA's x tile or W half tile (bf16)
constexpr int kRawBytes = 128 * kBK * 4;        // 32 KB: one CTA's fp32 x tile as loaded
constexpr int kConvThreads = 128;               // warps 2, 3, 8, 9

// operands: bf16 x bf16; fp32 x converted to bf16; e4m3 x e4m3 with bf16 x quantised in-kernel; e4m3 x e4m3 with x
// already e4m3 in memory (the output of an FP8 layer before it: both operands come straight through TMA)
enum : int { MODE_BF16 = 0, MODE_XF32 = 1, MODE_FP8 = 2, MODE_FP8Q = 3 };

template <int MODE>
struct Cfg {
  static constexpr bool kConv = MODE == MODE_XF32 || MODE == MODE_FP8;
  static constexpr bool kF8 = MODE == MODE_FP8 || MODE == MODE_FP8Q;
  static constexpr int kStages = kConv ? 4 : 6;
  static constexpr int kRawStages = kConv ? 2 : 0;
  static constexpr int kKStep = kF8 ? 128 : 64;   // elements of K per stage: one 128-byte row per operand row
  static constexpr int kSmemCtrl = 1024;
  static constexpr int kSmemTotal = kStages * 2 * kTileBytes + kRawStages * kRawBytes + kSmemCtrl + 1024;
  static_assert(kSmemTotal <= 232448, "exceeds the 227 KB shared memory of an sm_100 CTA");
};

struct __align__(16) Ctrl {
  uint64_t full[8], empty[8];
  uint64_t raw_full[2], raw_empty[2];
  uint64_t acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= 1024, "control block too large");

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
upr_linear_pair_kernel(const __grid_constant__ CUtensorMap tmap_x,   // box 128 rows x 64 k (bf16: SWIZZLE_128B; fp32: none)
                       const __grid_constant__ CUtensorMap tmap_w,   // bf16 [N, K], box 128 x 64, SWIZZLE_128B
                       const Args args) {
  using C = Cfg<MODE>;
  constexpr bool X_F32 = C::kConv;   // x goes through the converter warps
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_aligned = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t a_smem = smem_base;
  const uint32_t b_smem = a_smem + C::kStages * kTileBytes;
  const uint32_t raw_smem = b_smem + C::kStages * kTileBytes;
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_aligned + C::kStages * 2 * kTileBytes + C::kRawStages * kRawBytes);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = blockIdx.x & 1u;     // == %cluster_ctarank for cluster dims (2,1,1); warp-uniform to the compiler
  const bool leader = rank == 0;
  const int pair_id = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int m_tiles = static_cast<int>((args.M + kBM - 1) / kBM);
  const int n_tiles = (args.N + kBN - 1) / kBN;
  const int k_steps = args.K / C::kKStep;
  const long long total_tiles = static_cast<long long>(m_tiles) * n_tiles;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::kStages; ++i) {
      // leader's copy is used: its producer's arrive.expect_tx (bytes of both CTAs) and, for fp32 x, the four
      // converter warps of each CTA
      mbar_init(smem_u32(&ctrl->full[i]), X_F32 ? 9 : 1);
      mbar_init(smem_u32(&ctrl->empty[i]), 1);      // multicast commit
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl->raw_full[i]), 1);
      mbar_init(smem_u32(&ctrl->raw_empty[i]), 4);
      mbar_init(smem_u32(&ctrl->acc_full[i]), 1);   // multicast commit
      mbar_init(smem_u32(&ctrl->acc_empty[i]), 16); // 8 epilogue warps of each CTA (leader's copy)
    }
    fence_mbar_init();
  }
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmap_x);
    tma_prefetch_desc(&tmap_w);
  }
  if (warp == 1) {
    tmem_alloc_pair(smem_u32(&ctrl->tmem_base), 512);
    tmem_relinquish_pair();
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;

  if (warp == 0) {
    // ================================================================= producer (both CTAs)
    if (elect_one()) {
      const uint32_t lead_full = mapa_shared(smem_u32(&ctrl->full[0]), 0);
      uint32_t it = 0, raw_it = 0;
      for (long long t = pair_id; t < total_tiles; t += n_pairs) {
        const int mb = static_cast<int>(t / n_tiles), nb = static_cast<int>(t % n_tiles);
        const int xrow = mb * kBM + static_cast<int>(rank) * 128;     // this CTA's 128 rows of x
        const int wrow = nb * kBN + static_cast<int>(rank) * 128;     // ... and its half of the W tile
        for (int ks = 0; ks < k_steps; ++ks, ++it) {
          const uint32_t s = it % C::kStages, ph = (it / C::kStages) & 1;
          mbar_wait<1>(smem_u32(&ctrl->empty[s]), ph ^ 1);
          const uint32_t full = lead_full + s * 8;
          if (X_F32) {
            if (leader) mbar_arrive_expect_tx(smem_u32(&ctrl->full[s]), 2 * kTileBytes);
            tma_load_2d_pair(b_smem + s * kTileBytes, &tmap_w, ks * C::kKStep, wrow, full);
            const uint32_t rs = raw_it % 2, rph = (raw_it / 2) & 1;
            mbar_wait<2>(smem_u32(&ctrl->raw_empty[rs]), rph ^ 1);
            const uint32_t rfull = smem_u32(&ctrl->raw_full[rs]);
            mbar_arrive_expect_tx(rfull, kRawBytes);
            tma_load_2d(raw_smem + rs * kRawBytes, &tmap_x, ks * C::kKStep, xrow, rfull);
            ++raw_it;
          } else {
            if (leader) mbar_arrive_expect_tx(smem_u32(&ctrl->full[s]), 4 * kTileBytes);
            tma_load_2d_pair(a_smem + s * kTileBytes, &tmap_x, ks * C::kKStep, xrow, full);
            tma_load_2d_pair(b_smem + s * kTileBytes, &tmap_w, ks * C::kKStep, wrow, full);
          }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ================================================================= MMA issuer (leader)
    if (leader) {
      if (elect_one()) {
        constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO 1024, version 1, SWIZZLE_128B
        constexpr uint32_t kLoK = (16u >> 4) << 16;
        constexpr uint32_t kIdesc = C::kF8 ? make_idesc_e4m3(kBM, kBN) : make_idesc_bf16(kBM, kBN, 0, 0);
        auto mk_desc = [](uint32_t lo) {
          return (static_cast<uint64_t>(kDescHi) << 32) | static_cast<uint64_t>(lo);
        };
        const uint32_t a_lo = ((a_smem & 0x3FFFFu) >> 4) | kLoK;
        const uint32_t b_lo = ((b_smem & 0x3FFFFu) >> 4) | kLoK;
        uint32_t it = 0, n_acc = 0;
        for (long long t = pair_id; t < total_tiles; t += n_pairs, ++n_acc) {
          const uint32_t ab = n_acc & 1;
          if (n_acc >= 2) mbar_wait<3>(smem_u32(&ctrl->acc_empty[ab]), ((n_acc >> 1) - 1) & 1);
          tc_fence_after();
          for (int ks = 0; ks < k_steps; ++ks, ++it) {
            const uint32_t s = it % C::kStages, ph = (it / C::kStages) & 1;
            mbar_wait<4>(smem_u32(&ctrl->full[s]), ph);
            tc_fence_after();
#pragma unroll
            for (int k = 0; k < 4; ++k) {   // 32 bytes of K per instruction: 16 bf16 or 32 e4m3 elements
              const uint64_t da = mk_desc(a_lo + ((s * kTileBytes + k * 32) >> 4));
              const uint64_t db = mk_desc(b_lo + ((s * kTileBytes + k * 32) >> 4));
              if (C::kF8) umma_ss_pair_f8(tmem_base + ab * kBN, da, db, kIdesc, (ks > 0 || k > 0) ? 1u : 0u);
              else umma_ss_pair(tmem_base + ab * kBN, da, db, kIdesc, (ks > 0 || k > 0) ? 1u : 0u);
            }
            umma_commit_pair(smem_u32(&ctrl->empty[s]));
          }
          umma_commit_pair(smem_u32(&ctrl->acc_full[ab]));
        }
      }
    }
    __syncwarp();
  } else if (warp == 2 || warp == 3 || warp == 8 || warp == 9) {
    // ================================================================= converters (fp32 x / FP8), both CTAs
    if constexpr (X_F32) {
      const int ctid = (warp < 4 ? warp - 2 : warp - 6) * 32 + lane;   // 0..127
      const uint32_t lead_full = mapa_shared(smem_u32(&ctrl->full[0]), 0);
      uint32_t it = 0;
      for (long long t = pair_id; t < total_tiles; t += n_pairs) {
        for (int ks = 0; ks < k_steps; ++ks, ++it) {
          const uint32_t s = it % C::kStages, ph = (it / C::kStages) & 1;
          const uint32_t rs = it % 2, rph = (it / 2) & 1;
          mbar_wait<5>(smem_u32(&ctrl->empty[s]), ph ^ 1);      // the MMA has finished with this stage's x tile
          mbar_wait<6>(smem_u32(&ctrl->raw_full[rs]), rph);
          const uint32_t raw = raw_smem + rs * kRawBytes;
          const uint32_t tile = a_smem + s * kTileBytes;
          if constexpr (MODE == MODE_FP8) {
            // raw: 128 rows x 128 bf16 (256 B per row) -> 128 rows x 128 e4m3 (one swizzled 128-byte row each);
            // byte = cvt.rn.satfinite.e4m3(x * x_mult), the product rounded once in fp32
#pragma unroll 4
            for (int p = ctid; p < 128 * 8; p += kConvThreads) {
              const int row = p >> 3, c16 = p & 7;                 // 16 bf16 -> one 16-byte e4m3 chunk
              const uint4 a = lds128(raw + row * 256 + c16 * 32), b = lds128(raw + row * 256 + c16 * 32 + 16);
              const uint32_t in[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
              uint32_t o[4];
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const float f0 = __uint_as_float(in[2 * k] << 16) * args.x_mult;
                const float f1 = __uint_as_float(in[2 * k] & 0xffff0000u) * args.x_mult;
                const float f2 = __uint_as_float(in[2 * k + 1] << 16) * args.x_mult;
                const float f3 = __uint_as_float(in[2 * k + 1] & 0xffff0000u) * args.x_mult;
                o[k] = static_cast<uint32_t>(__nv_cvt_float2_to_fp8x2(make_float2(f0, f1), __NV_SATFINITE, __NV_E4M3)) |
                       (static_cast<uint32_t>(__nv_cvt_float2_to_fp8x2(make_float2(f2, f3), __NV_SATFINITE, __NV_E4M3)) << 16);
              }
              sts128(tile + row * 128 + ((c16 ^ (row & 7)) << 4), o[0], o[1], o[2], o[3]);
            }
          } else {
#pragma unroll 4
          for (int p = ctid; p < 128 * 8; p += kConvThreads) {
            const int row = p >> 3, c8 = p & 7;                  // 8 floats -> one 16-byte bf16 chunk
            const uint4 a = lds128(raw + row * 256 + c8 * 32), b = lds128(raw + row * 256 + c8 * 32 + 16);
            sts128(tile + row * 128 + ((c8 ^ (row & 7)) << 4),
                   pack_bf16x2(__uint_as_float(a.x), __uint_as_float(a.y)),
                   pack_bf16x2(__uint_as_float(a.z), __uint_as_float(a.w)),
                   pack_bf16x2(__uint_as_float(b.x), __uint_as_float(b.y)),
                   pack_bf16x2(__uint_as_float(b.z), __uint_as_float(b.w)));
          }
          }
          fence_proxy_async_smem();   // generic-proxy tile writes -> visible to tcgen05.mma
          __syncwarp();
          if (lane == 0) {
            mbar_arrive(smem_u32(&ctrl->raw_empty[rs]));
            mbar_arrive_cluster(lead_full + s * 8);
          }
        }
      }
    }
  } else {
    // ================================================================= epilogue (both CTAs)
    // two groups of four warps: warps 4-7 take the accumulator's columns [0, 128), warps 10-13 [128, 256) -- with
    // a fused activation the epilogue of a 256-column tile is otherwise slower than the tile's MMAs
    const int ew = warp & 3;                                   // TMEM lane quarter (== warp % 4)
    const int ehalf = warp >= 10 ? 1 : 0;
    const uint32_t lane_base = static_cast<uint32_t>(ew * 32) << 16;
    const uint32_t lead_acc_empty = mapa_shared(smem_u32(&ctrl->acc_empty[0]), 0);
    uint32_t n_acc = 0;
    for (long long t = pair_id; t < total_tiles; t += n_pairs, ++n_acc) {
      const int mb = static_cast<int>(t / n_tiles), nb = static_cast<int>(t % n_tiles);
      const uint32_t ab = n_acc & 1;
      mbar_wait<7>(smem_u32(&ctrl->acc_full[ab]), (n_acc >> 1) & 1);
      tc_fence_after();
      const long long row = static_cast<long long>(mb) * kBM + rank * 128 + ew * 32 + lane;
      const bool row_ok = row < args.M;
      // pool mode: first pool row of this token's slot (head 0), or -1
      long long kv_row0 = -1;
      if (args.tok_slot != nullptr && row_ok)
        kv_row0 = ((static_cast<long long>(args.kv_layer) * args.kv_S + __ldg(args.tok_slot + row)) * args.kv_H) * args.kv_n +
                  __ldg(args.tok_pos + row);
      // one 32-column chunk: + bias, activation, + residual, store (activation as a compile-time branch)
      auto chunk = [&](auto act_tag, const int c0) {
        constexpr int kAct = decltype(act_tag)::value;
        uint32_t r[32];
        tmem_ld32(tmem_base + lane_base + ab * kBN + c0, r);
        tmem_wait_ld_regs(r);
        if (c0 + 32 == (ehalf + 1) * (kBN / 2)) {   // this warp's last chunk is in registers
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(lead_acc_empty + ab * 8);
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
          if (C::kF8) {
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] *= args.out_scale;
          }
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
            const int col = col0 + c, h = col / args.kv_d, tt = col - h * args.kv_d;   // 8 columns stay inside one head
            __nv_bfloat16* dst = static_cast<__nv_bfloat16*>(args.y) +
                                 (kv_row0 + static_cast<long long>(h) * args.kv_n) * args.kv_d + tt;
            *reinterpret_cast<uint4*>(dst) = make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]),
                                                        pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
          } else if (C::kF8 && args.y_is_fp8) {
            // the next FP8 layer's operand: byte = cvt.rn.satfinite.e4m3(value * y_mult), product rounded once in fp32
            uint32_t o[2];
#pragma unroll
            for (int k = 0; k < 2; ++k)
              o[k] = static_cast<uint32_t>(__nv_cvt_float2_to_fp8x2(
                         make_float2(v[4 * k] * args.y_mult, v[4 * k + 1] * args.y_mult), __NV_SATFINITE, __NV_E4M3)) |
                     (static_cast<uint32_t>(__nv_cvt_float2_to_fp8x2(
                          make_float2(v[4 * k + 2] * args.y_mult, v[4 * k + 3] * args.y_mult), __NV_SATFINITE, __NV_E4M3))
                      << 16);
            *reinterpret_cast<uint2*>(static_cast<uint8_t*>(args.y) + row * args.N + col0 + c) = make_uint2(o[0], o[1]);
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
      for (int c0 = ehalf * (kBN / 2); c0 < (ehalf + 1) * (kBN / 2); c0 += 32) {
        if (args.act == ACT_SILU) chunk(cuda::std::integral_constant<int, ACT_SILU>{}, c0);
        else if (args.act == ACT_RELU) chunk(cuda::std::integral_constant<int, ACT_RELU>{}, c0);
        else chunk(cuda::std::integral_constant<int, ACT_NONE>{}, c0);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync_all();      // the peer may still signal this CTA's barriers
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base, 512);
  }
}

}  // namespace lin2
}  // namespace upr
