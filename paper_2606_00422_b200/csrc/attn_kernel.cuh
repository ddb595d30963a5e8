// attn_kernel.cuh -- ranking-head cross-attention forward (steps a2-a7 of SURVEY.md 8(a)).
//
// For each user b, candidate rows q[c] (cand_offsets[b] <= c < cand_offsets[b+1]) attend over
// that user's cached history K/V rows [0, L_b) -- never over other candidates (PAPER.md:138,
// 198); optionally each candidate also sees its own key/value (identity block of the
// M-FALCON mask).  out = softmax(scale * q K^T) V, fp32.
//
// Persistent, warp-specialised CTA (one per SM, 512 threads), work item = (layer, user, head,
// history split, block of <= 256 candidates):
//   warps 0-3   : softmax group for candidate tile 0 (rows   0..127), one thread per row
//   warps 4-7   : softmax group for candidate tile 1 (rows 128..255)
//   warp  8     : scheduler + producer (decodes work items from the device offset tables and
//                 streams the user's K/V tiles HBM -> smem, once per item: TMA tensor boxes
//                 for a bf16 cache, contiguous bulk copies of raw rows for fp8 / fp32 caches)
//   warp  9     : tcgen05.mma issuer: S_t = Q_t K^T (SS), O_t += P_t V (A = P from TMEM)
//   warps 10-11 : converters (fp8 / fp32 caches only): raw rows -> bf16 swizzled MMA tiles,
//                 "dequantised in registers"; the scales fold into the softmax scale (K) and
//                 the epilogue (V), so the conversion is a pure, exact type change for E4M3
//   warps 12-15 : epilogue group: drains O_t from TMEM, scales by 1/l, transposes 32x32
//                 blocks through padded shared memory and writes full 128-byte lines, while
//                 the softmax and MMA warps are already on the next item
// TMEM (512 cols): S0 [0,128) S1 [128,256) O0 [256,256+D) O1 [256+D,256+2D); P_t (bf16)
// overwrites the first 64 columns of S_t once S_t has been read into registers.
// Online softmax in fp32 with lazy rescaling of O (only when the running max grows by more
// than 2^8); row reductions are thread-local because the 32x32b TMEM load gives each thread
// a whole row.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <cuda/std/type_traits>

#include "ptx.cuh"

namespace upr {

constexpr int kTileM = 128;     // candidate rows per MMA tile == TMEM lanes
constexpr int kTileN = 128;     // keys per K/V smem tile
constexpr int kNB = 2;          // S buffers per candidate tile
constexpr int kSubN = kTileN / kNB;   // keys per softmax / MMA step: S(s + kNB) is issued behind PV(s)
constexpr int kQBlock = 256;    // candidate rows per work item (two tiles)
constexpr int kRowAlign = 16;   // UPR_ROW_ALIGN
constexpr int kAttnThreads = 512;     // 2 softmax warpgroups + {TMA, MMA, 2 converters} + epilogue
// setmaxnreg budgets.  The pool is what the CTA was given at launch (512 threads x 128
// registers), not the whole register file: an .inc beyond it blocks forever.
constexpr int kLaunchRegs = 128;
constexpr int kSoftmaxRegs = 168;    //   2 softmax warpgroups
constexpr int kOtherRegs = 56;       //   producer / MMA / converter warpgroup
constexpr int kEpilogueRegs = 88;    //   epilogue warpgroup
static_assert(256 * kSoftmaxRegs + 128 * kOtherRegs + 128 * kEpilogueRegs <= kAttnThreads * kLaunchRegs,
              "setmaxnreg budgets exceed the CTA's register allocation");
constexpr int kProducerWarp = 8;
constexpr int kMmaWarp = 9;
constexpr int kConvWarp0 = 10;        // warps 10, 11
constexpr int kConvThreads = 64;
constexpr int kEpiWarp0 = 12;         // warps 12..15
constexpr int kTmemCols = 512;
constexpr float kRescaleTau = 8.0f;  // lazy-rescale threshold, log2 units
constexpr int kEpiRowBytes = 144;     // 32 floats + 16 B pad: conflict-free 16-byte accesses
// (a warp's staging block is 32 x 144 B = 4608 B; the TMA-store path uses its first 4096 B as a
// dense, 128-byte-swizzled 32 x 32 fp32 box, so the block must start on a 1024-byte boundary)

enum : int { KV_BF16 = 0, KV_FP8 = 1, KV_F32 = 2 };

struct AttnArgs {
  const void* q;
  const void* k_self;
  const void* v_self;
  float* out;
  const int32_t* seq_lens;
  const int32_t* cand_offsets;
  const float* k_scale;
  const float* v_scale;
  const uint8_t* k_raw;   // fp8 / fp32 caches: base of the packed cache (bulk-copied raw rows)
  const uint8_t* v_raw;
  float* part_o;          // split-K partial O~  [n_layers][total_q][H][ns][D]
  float* part_ml;         // split-K partial (m, l) [n_layers][total_q][H][ns][2]
  unsigned int* counter;  // dynamic work counter (zeroed before launch) or nullptr = static
  const int32_t* slot_ids;  // non-null: K/V are read in place from the pool [n_layers, pool_S, H, pool_n, D]
  int pool_S, pool_n;
  int B, H, n_layers, num_splits;
  int q_is_f32;
  int scale_per_user;     // FP8 scales indexed [layer, user, head] instead of [layer, head]
  int q_tma;              // 1: tmap_q describes `q` as [n_layers*total_q, H*D] bf16: the producer loads Q tiles by TMA
  int out_tma;            // 1: tmap_out describes `out` as [n_layers*total_q, H*D] fp32 (full tiles use TMA stores)
  float scale_log2;       // sm_scale * log2(e)
};

struct WorkItem {
  int valid;     // 0 = no more work
  int layer, h, split;
  int q_row0;    // first candidate row (global index into [total_q]) of this block
  int n_rows;    // valid rows in this block (1..256)
  int kv_row0;   // row into the 2-D [n_layers*H*R, d] cache view of the first key of the split
  int key0;      // first key index (within the user) of this split
  int n_keys;    // valid keys in this split's range (>= 0)
  int total_q;   // cand_offsets[B]
  int b;         // user
};

template <int D, int KV>
struct AttnCfg {
  static constexpr int kBoxBytes = kTileN * 128;            // one [128 rows x 64 bf16] box
  static constexpr int kBoxes = D / 64;                     // boxes per tile
  static constexpr int kTileBytes = kBoxBytes * kBoxes;     // Q tile, K tile or V tile (bf16)
  static constexpr int kStages =                            // K/V ring slots (bf16 tiles)
      (KV == KV_BF16) ? ((D == 128) ? 4 : 8) : ((D == 128) ? 3 : 6);
  // raw ring (fp8 / fp32 caches): one slot = kRawRows contiguous cache rows
  static constexpr int kElemBytes = (KV == KV_FP8) ? 1 : (KV == KV_F32) ? 4 : 2;
  static constexpr int kRawRows = (KV == KV_F32) ? 32 : 128;
  static constexpr int kRawSlotBytes = kRawRows * D * kElemBytes;   // 16 KB (D=128) / 8 KB
  static constexpr int kRawStages = (KV == KV_BF16) ? 0 : ((D == 128) ? 2 : 4);
  static constexpr int kRawPerTile = kTileN / kRawRows;
  static constexpr int kSmemQ = 2 * kTileBytes;
  static constexpr int kSmemKV = kStages * kTileBytes;
  static constexpr int kSmemRaw = kRawStages * kRawSlotBytes;
  static constexpr int kEpiWarpBytes = 5120;                // 32 x 144 B rounded up to 1024
  static constexpr int kSmemEpi = 4 * kEpiWarpBytes;        // one 32 x 32 fp32 block per warp
  static constexpr int kSmemCtrl = 6144;
  static constexpr int kSmemTotal =
      kSmemQ + kSmemKV + kSmemRaw + kSmemEpi + kSmemCtrl + 1024;  // + alignment slack
  // FP8 caches multiply in fp16 (Q converted on the way into shared memory, K / V from E4M3 by one cvt per two
  // bytes, P packed as fp16): every E4M3 value and every weight <= 2^8 is representable, and the converter warps
  // need a quarter of the instructions of the bf16 route.  bf16 / fp32 caches multiply in bf16.
  static constexpr bool kF16 = (KV == KV_FP8);
  static constexpr uint32_t kIdescQK = kF16 ? make_idesc_f16(kTileM, kSubN, 0, 0) : make_idesc_bf16(kTileM, kSubN, 0, 0);
  static constexpr uint32_t kIdescPV = kF16 ? make_idesc_f16(kTileM, D, 0, 1) : make_idesc_bf16(kTileM, D, 0, 1);
  static_assert(kSmemTotal <= 232448, "exceeds the 227 KB shared memory of an sm_100 CTA");
};

struct __align__(16) AttnCtrl {
  uint64_t kv_full[8];
  uint64_t kv_empty[8];
  uint64_t raw_full[4];
  uint64_t raw_empty[4];
  uint64_t q_full[2];
  uint64_t q_empty[2];     // the item's last S MMA of tile t has read Q_t (TMA Q loads only)
  uint64_t s_full[2][2];   // [tile][S buffer]
  uint64_t p_full[2][2];
  uint64_t pv_done[2];     // one completion per PV sub-tile MMA of tile t
  uint64_t o_full[2];
  uint64_t o_empty[2];
  uint64_t l_ready[2];
  uint64_t item_full[2];
  uint64_t item_empty[2];
  WorkItem items[2];
  uint32_t tmem_base;
  uint32_t pad_[3];
  float epi_inv[2][2][kTileM];    // [item slot][tile][row]: 1/l (or 1 for split-K partials)
  float epi_wself[2][2][kTileM];  // weight of the candidate's own value row
};
static_assert(sizeof(AttnCtrl) <= 6144, "control block too large");

// ---------------------------------------------------------------------------------------
// Scheduler state: a forward-only cursor over users, 32 at a time (one per lane).
// ---------------------------------------------------------------------------------------
struct UserCursor {
  int b0;           // first user of the current 32-user window
  int w_before;     // work items of users < b0 (within one layer)
  int rows_before;  // aligned cache rows of users < b0
};

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

// items and aligned rows of user u (0 if u >= B)
__device__ __forceinline__ void user_sizes(const AttnArgs& a, int u, int& w, int& rows, int& C,
                                           int& L) {
  w = 0; rows = 0; C = 0; L = 0;
  if (u < a.B) {
    int c0 = __ldg(a.cand_offsets + u), c1 = __ldg(a.cand_offsets + u + 1);
    C = c1 - c0;
    L = __ldg(a.seq_lens + u);
    int nq = (C + kQBlock - 1) / kQBlock;
    w = nq * a.H * a.num_splits;
    rows = (L + kRowAlign - 1) / kRowAlign * kRowAlign;
  }
}

// ---------------------------------------------------------------------------------------
// Q tile: global [rows, H*D] (bf16 or fp32) -> bf16 smem in the 128B-swizzled K-major layout
// the UMMA descriptor expects (identical to what a SWIZZLE_128B TMA box would write).
// ---------------------------------------------------------------------------------------
template <int D, bool kToF16 = false>
__device__ __forceinline__ void load_q_tile(uint32_t tile_smem, const void* q, bool q_is_f32,
                                            size_t elem_base, size_t row_stride, int rows_valid,
                                            int tid128) {
  constexpr int CPR = D / 8;  // 16-byte bf16 chunks per row
#pragma unroll 4
  for (int i = 0; i < CPR; ++i) {
    int id = i * 128 + tid128;
    int row = id / CPR, c = id % CPR;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (row < rows_valid) {
      size_t e = elem_base + static_cast<size_t>(row) * row_stride + static_cast<size_t>(c) * 8;
      if (!q_is_f32) {
        v = __ldg(reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(q) + e));
        if (kToF16) {   // bf16 -> fp16 (exact for |x| in fp16's normal range; saturating beyond it)
          v.x = pack_f16x2(__uint_as_float(v.x << 16), __uint_as_float(v.x & 0xffff0000u));
          v.y = pack_f16x2(__uint_as_float(v.y << 16), __uint_as_float(v.y & 0xffff0000u));
          v.z = pack_f16x2(__uint_as_float(v.z << 16), __uint_as_float(v.z & 0xffff0000u));
          v.w = pack_f16x2(__uint_as_float(v.w << 16), __uint_as_float(v.w & 0xffff0000u));
        }
      } else {
        const float4* p = reinterpret_cast<const float4*>(static_cast<const float*>(q) + e);
        float4 a = __ldg(p), b = __ldg(p + 1);
        v.x = kToF16 ? pack_f16x2(a.x, a.y) : pack_bf16x2(a.x, a.y);
        v.y = kToF16 ? pack_f16x2(a.z, a.w) : pack_bf16x2(a.z, a.w);
        v.z = kToF16 ? pack_f16x2(b.x, b.y) : pack_bf16x2(b.x, b.y);
        v.w = kToF16 ? pack_f16x2(b.z, b.w) : pack_bf16x2(b.z, b.w);
      }
    }
    int box = c >> 3, cc = c & 7;
    uint32_t addr = tile_smem + box * (kTileM * 128) + row * 128 + ((cc ^ (row & 7)) << 4);
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y),
                 "r"(v.z), "r"(v.w)
                 : "memory");
  }
}

// Same tile, bf16 source, through cp.async (LDGSTS): no register staging, all 16-byte copies
// of the thread in flight at once; rows >= rows_valid are zero-filled (src-size 0).
template <int D>
__device__ __forceinline__ void load_q_tile_async(uint32_t tile_smem, const void* q,
                                                  size_t elem_base, size_t row_stride,
                                                  int rows_valid, int tid128) {
  constexpr int CPR = D / 8;
  const __nv_bfloat16* qb = static_cast<const __nv_bfloat16*>(q);
#pragma unroll
  for (int i = 0; i < CPR; ++i) {
    const int id = i * 128 + tid128;
    const int row = id / CPR, c = id % CPR;
    const bool ok = row < rows_valid;
    const __nv_bfloat16* src =
        qb + elem_base + static_cast<size_t>(ok ? row : 0) * row_stride + static_cast<size_t>(c) * 8;
    const int box = c >> 3, cc = c & 7;
    const uint32_t dst = tile_smem + box * (kTileM * 128) + row * 128 + ((cc ^ (row & 7)) << 4);
    cp_async_16(dst, src, ok ? 16u : 0u);
  }
  cp_async_commit();
}

// dot(q_row, kself_row) for the self logit; both rows in global, bf16 or fp32
template <int D>
__device__ __forceinline__ float row_dot(const void* a, const void* b, bool is_f32, size_t e) {
  float acc = 0.f;
  if (!is_f32) {
    const uint4* pa = reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(a) + e);
    const uint4* pb = reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(b) + e);
#pragma unroll 4
    for (int i = 0; i < D / 8; ++i) {
      uint4 x = __ldg(pa + i), y = __ldg(pb + i);
      const __nv_bfloat162* xs = reinterpret_cast<const __nv_bfloat162*>(&x);
      const __nv_bfloat162* ys = reinterpret_cast<const __nv_bfloat162*>(&y);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        float2 fx = __bfloat1622float2(xs[k]), fy = __bfloat1622float2(ys[k]);
        acc = fmaf(fx.x, fy.x, acc);
        acc = fmaf(fx.y, fy.y, acc);
      }
    }
  } else {
    const float4* pa = reinterpret_cast<const float4*>(static_cast<const float*>(a) + e);
    const float4* pb = reinterpret_cast<const float4*>(static_cast<const float*>(b) + e);
#pragma unroll 4
    for (int i = 0; i < D / 4; ++i) {
      float4 x = __ldg(pa + i), y = __ldg(pb + i);
      acc = fmaf(x.x, y.x, acc);
      acc = fmaf(x.y, y.y, acc);
      acc = fmaf(x.z, y.z, acc);
      acc = fmaf(x.w, y.w, acc);
    }
  }
  return acc;
}

// ---------------------------------------------------------------------------------------
// The kernel
// ---------------------------------------------------------------------------------------
template <int D, int KV>
__global__ void __launch_bounds__(kAttnThreads, 1)
upr_attn_fwd_kernel(const __grid_constant__ CUtensorMap tmap_k,
                    const __grid_constant__ CUtensorMap tmap_v,
                    const __grid_constant__ CUtensorMap tmap_out,
                    const __grid_constant__ CUtensorMap tmap_q, const AttnArgs args) {
  using Cfg = AttnCfg<D, KV>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_aligned = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t q_smem = smem_base;
  const uint32_t kv_smem = q_smem + Cfg::kSmemQ;
  const uint32_t raw_smem = kv_smem + Cfg::kSmemKV;
  const uint32_t epi_smem = raw_smem + Cfg::kSmemRaw;
  AttnCtrl* ctrl = reinterpret_cast<AttnCtrl*>(smem_aligned + Cfg::kSmemQ + Cfg::kSmemKV +
                                               Cfg::kSmemRaw + Cfg::kSmemEpi);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  constexpr bool kConvert = (KV != KV_BF16);
  // arrivals that release an item slot: 256 softmax threads, MMA lane 0, one lane of each
  // epilogue warp, one lane of each converter warp
  constexpr uint32_t kItemReaders = 256 + 1 + 4 + (kConvert ? 2 : 0);
  // bf16 caches with a host-known total_q: Q tiles arrive by TMA, issued by the producer as soon
  // as the previous item's last S MMA has released the tile (the cp.async path of the softmax
  // warps could only start one step before the item's end and its latency showed at every item)
  const bool q_by_tma = !kConvert && args.q_tma != 0;

  // ------------------------------------------------------------------ one-time setup
  // diagnostic: SM cycles and nanoseconds this CTA lives, left in the workspace's counter block (words 16..19) by
  // CTA 0 -- their ratio is the clock the SMs really ran at under this kernel (bench.py reports it)
  unsigned long long diag_t0 = 0, diag_c0 = 0;
  const bool diag = blockIdx.x == 0 && threadIdx.x == 0 && args.counter != nullptr;
  if (diag) {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(diag_t0));
    diag_c0 = static_cast<unsigned long long>(clock64());
  }
  if (threadIdx.x == 0) {
    for (int i = 0; i < Cfg::kStages; ++i) {
      mbar_init(smem_u32(&ctrl->kv_full[i]), kConvert ? kConvThreads : 1);
      mbar_init(smem_u32(&ctrl->kv_empty[i]), 1);
    }
    for (int i = 0; i < Cfg::kRawStages; ++i) {
      mbar_init(smem_u32(&ctrl->raw_full[i]), 1);
      mbar_init(smem_u32(&ctrl->raw_empty[i]), kConvThreads);
    }
    for (int t = 0; t < 2; ++t) {
      mbar_init(smem_u32(&ctrl->q_full[t]), q_by_tma ? 1 : 4);   // TMA transaction / one arrival per softmax warp
      mbar_init(smem_u32(&ctrl->q_empty[t]), 1);
      for (int bf = 0; bf < 2; ++bf) {
        mbar_init(smem_u32(&ctrl->s_full[t][bf]), 1);
        mbar_init(smem_u32(&ctrl->p_full[t][bf]), 4);
      }
      mbar_init(smem_u32(&ctrl->pv_done[t]), 1);
      mbar_init(smem_u32(&ctrl->o_full[t]), 1);
      mbar_init(smem_u32(&ctrl->o_empty[t]), 4);
      mbar_init(smem_u32(&ctrl->l_ready[t]), 4);
      mbar_init(smem_u32(&ctrl->item_full[t]), 1);
      mbar_init(smem_u32(&ctrl->item_empty[t]), kItemReaders);
    }
    fence_mbar_init();
  }
  if (warp == kProducerWarp && !kConvert) {
    if (lane == 0) {
      tma_prefetch_desc(&tmap_k);
      tma_prefetch_desc(&tmap_v);
    }
  }
  if (warp == kMmaWarp) {
    tmem_alloc(smem_u32(&ctrl->tmem_base), kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;

  if (warp == kProducerWarp) {
    // ================================================================= scheduler + producer
    setmaxnreg_dec<kOtherRegs>();
    // one pass over the users: items per layer (W) and aligned rows per (layer, head) (R)
    int W = 0, R = 0;
    for (int u0 = 0; u0 < args.B; u0 += 32) {
      int w, rows, C, L;
      user_sizes(args, u0 + lane, w, rows, C, L);
      W += w;
      R += rows;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      W += __shfl_xor_sync(0xffffffffu, W, o);
      R += __shfl_xor_sync(0xffffffffu, R, o);
    }
    const int total_items = W * args.n_layers;
    const int total_q = (args.B > 0) ? __ldg(args.cand_offsets + args.B) : 0;

    UserCursor cur{0, 0, 0};
    uint32_t q_uses[2] = {0, 0};   // Q tile loads issued so far, per tile (TMA Q loads)
    uint32_t kv_it = 0;   // bf16 ring position (TMA mode) / raw ring position (convert mode)
    for (uint32_t n = 0;; ++n) {
      const int islot = n & 1;
      mbar_wait<1>(smem_u32(&ctrl->item_empty[islot]), ((n >> 1) & 1) ^ 1);
      int idx;
      if (args.counter != nullptr) {
        idx = 0;
        if (lane == 0) idx = static_cast<int>(atomicAdd(args.counter, 1u));
        idx = __shfl_sync(0xffffffffu, idx, 0);
      } else {
        idx = static_cast<int>(blockIdx.x + n * gridDim.x);
      }
      if (idx >= total_items) {
        if (lane == 0) {
          ctrl->items[islot].valid = 0;
          mbar_arrive(smem_u32(&ctrl->item_full[islot]));
        }
        break;
      }
      const int layer = idx / W;
      const int r = idx - layer * W;
      if (r < cur.w_before) cur = UserCursor{0, 0, 0};
      // advance the window until it contains item r
      int w, rows, C, L, w_incl, rows_incl;
      for (;;) {
        user_sizes(args, cur.b0 + lane, w, rows, C, L);
        w_incl = warp_incl_scan(w, lane);
        rows_incl = warp_incl_scan(rows, lane);
        int w_tot = __shfl_sync(0xffffffffu, w_incl, 31);
        if (r < cur.w_before + w_tot) break;
        cur.w_before += w_tot;
        cur.rows_before += __shfl_sync(0xffffffffu, rows_incl, 31);
        cur.b0 += 32;
      }
      const unsigned hit = __ballot_sync(0xffffffffu, cur.w_before + w_incl > r);
      const int src = __ffs(hit) - 1;
      const int local = r - (cur.w_before + __shfl_sync(0xffffffffu, w_incl - w, src));
      const int row_off_b = cur.rows_before + __shfl_sync(0xffffffffu, rows_incl - rows, src);
      const int Cb = __shfl_sync(0xffffffffu, C, src);
      const int Lb = __shfl_sync(0xffffffffu, L, src);
      const int b = cur.b0 + src;
      const int nq = (Cb + kQBlock - 1) / kQBlock;
      const int per_h = nq * args.num_splits;
      const int h = local / per_h;
      const int rem = local - h * per_h;
      const int split = rem / nq;
      const int qblk = rem - split * nq;
      const int nt_user = (Lb + kTileN - 1) / kTileN;
      const int t0 = static_cast<int>((static_cast<long long>(split) * nt_user) / args.num_splits);
      const int t1 =
          static_cast<int>((static_cast<long long>(split + 1) * nt_user) / args.num_splits);
      const int key0 = t0 * kTileN;
      const int n_keys = (t1 > t0) ? (min(Lb, t1 * kTileN) - key0) : 0;
      // base row of the (layer, user, head) block in the 2-D [rows, d] view of the K/V storage:
      // packed cache [n_layers, H, R, d], or the pool itself [n_layers, S, H, n, d] (zero copy)
      const int kv_row0 =
          (args.slot_ids != nullptr)
              ? ((layer * args.pool_S + __ldg(args.slot_ids + b)) * args.H + h) * args.pool_n + key0
              : (layer * args.H + h) * R + row_off_b + key0;
      if (elect_one()) {
        WorkItem& it = ctrl->items[islot];
        it.valid = 1;
        it.layer = layer;
        it.h = h;
        it.split = split;
        it.q_row0 = __ldg(args.cand_offsets + b) + qblk * kQBlock;
        it.n_rows = min(kQBlock, Cb - qblk * kQBlock);
        it.kv_row0 = kv_row0;
        it.key0 = key0;
        it.n_keys = n_keys;
        it.total_q = total_q;
        it.b = b;
        mbar_arrive(smem_u32(&ctrl->item_full[islot]));
        // stream this item's K/V tiles: K0 V0 K1 V1 ...
        const int nt = (n_keys + kTileN - 1) / kTileN;
        // ... and its Q tiles, each as soon as the tile buffer is free again
        bool pendq[2] = {false, false};
        if (q_by_tma && nt > 0) {
          pendq[0] = true;
          pendq[1] = it.n_rows > kTileM;
        }
        auto try_issue_q = [&]() {
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            if (!pendq[t]) continue;
            if (q_uses[t] > 0 && !mbar_test(smem_u32(&ctrl->q_empty[t]), (q_uses[t] - 1) & 1)) continue;
            const uint32_t full = smem_u32(&ctrl->q_full[t]);
            mbar_arrive_expect_tx(full, Cfg::kTileBytes);
            const int qrow = layer * total_q + it.q_row0 + t * kTileM;
#pragma unroll
            for (int bx = 0; bx < Cfg::kBoxes; ++bx)
              tma_load_2d(q_smem + t * Cfg::kTileBytes + bx * Cfg::kBoxBytes, &tmap_q, h * D + bx * 64, qrow,
                          full);
            ++q_uses[t];
            pendq[t] = false;
          }
        };
        try_issue_q();
        for (int j = 0; j < nt; ++j) {
#pragma unroll
          for (int kv = 0; kv < 2; ++kv) {
            if constexpr (!kConvert) {
              const uint32_t slot = kv_it % Cfg::kStages;
              const uint32_t ph = (kv_it / Cfg::kStages) & 1;
              while (!mbar_try_wait<2>(smem_u32(&ctrl->kv_empty[slot]), ph ^ 1)) try_issue_q();
              const uint32_t full = smem_u32(&ctrl->kv_full[slot]);
              mbar_arrive_expect_tx(full, Cfg::kTileBytes);
              const uint32_t dst = kv_smem + slot * Cfg::kTileBytes;
#pragma unroll
              for (int bx = 0; bx < Cfg::kBoxes; ++bx)
                tma_load_2d(dst + bx * Cfg::kBoxBytes, kv == 0 ? &tmap_k : &tmap_v, bx * 64,
                            kv_row0 + j * kTileN, full);
              ++kv_it;
            } else {
              const uint8_t* base = (kv == 0) ? args.k_raw : args.v_raw;
#pragma unroll 1
              for (int c = 0; c < Cfg::kRawPerTile; ++c) {
                const uint32_t slot = kv_it % Cfg::kRawStages;
                const uint32_t ph = (kv_it / Cfg::kRawStages) & 1;
                mbar_wait<3>(smem_u32(&ctrl->raw_empty[slot]), ph ^ 1);
                const uint32_t full = smem_u32(&ctrl->raw_full[slot]);
                mbar_arrive_expect_tx(full, Cfg::kRawSlotBytes);
                const size_t row = static_cast<size_t>(kv_row0) + j * kTileN + c * Cfg::kRawRows;
                bulk_load_1d(raw_smem + slot * Cfg::kRawSlotBytes,
                             base + row * (D * Cfg::kElemBytes), Cfg::kRawSlotBytes, full);
                ++kv_it;
              }
            }
          }
        }
        while (pendq[0] || pendq[1]) try_issue_q();
      }
      __syncwarp();
    }
  } else if (warp == kMmaWarp) {
    // ================================================================= MMA issuer
    // Keys are processed in sub-tiles of 64 (two per 128-key smem tile).  Each candidate tile
    // t owns two 64-column S buffers, so S(s+2) is issued right behind PV(s) -- i.e. S(s+1) is
    // being computed while the softmax group works on S(s): the softmax warps do not wait for
    // the tensor pipe in steady state.  P(s) aliases the first 32 columns of S buffer s & 1.
    //
    // The whole role runs in ONE elected thread: inside an elect.sync region the compiler
    // knows every value is warp-uniform and builds descriptors on the uniform datapath (with
    // a plain lane test it wraps each tcgen05.mma in a R2UR waterfall loop), and there is no
    // reconvergence or warp-sync traffic on what is the serial critical path of the CTA.
    setmaxnreg_dec<kOtherRegs>();
    if (elect_one()) {
      uint32_t kv_pos = 0;                       // ring position of the next item's K tile 0
      uint32_t q_ph = 0, od_ph = 0, pf_ph = 0;   // phase bits: q_full[t], o_empty[t], p_full[t][buf]
      // descriptor words: lo = addr >> 4 | (LBO >> 4) << 16, hi = SBO >> 4 | version 1 | SWIZZLE_128B
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
      constexpr uint32_t kLoKmajor = (16u >> 4) << 16;                                     // Q, K
      constexpr uint32_t kLoMNmajor = (static_cast<uint32_t>(Cfg::kBoxBytes) >> 4) << 16;  // V
      auto mk_desc = [](uint32_t lo) {
        return (static_cast<uint64_t>(kDescHi) << 32) | static_cast<uint64_t>(lo);
      };
      const uint32_t q_lo = ((q_smem & 0x3FFFFu) >> 4) | kLoKmajor;
      const uint32_t kv_lo = (kv_smem & 0x3FFFFu) >> 4;
      const uint32_t bar_s = smem_u32(&ctrl->s_full[0][0]);    // [t][buf] -> + (2t + buf) * 8
      const uint32_t bar_p = smem_u32(&ctrl->p_full[0][0]);
      for (uint32_t n = 0;; ++n) {
        const int islot = n & 1;
        mbar_wait<4>(smem_u32(&ctrl->item_full[islot]), (n >> 1) & 1);
        if (!ctrl->items[islot].valid) break;
        const int n_keys = ctrl->items[islot].n_keys;
        const int nt = (n_keys + kTileN - 1) / kTileN;
        const int nsub = (n_keys + kSubN - 1) / kSubN;
        const int ntile = (ctrl->items[islot].n_rows > kTileM) ? 2 : 1;
        if (nsub > 0) {
#pragma unroll
          for (int t = 0; t < 2; ++t)
            if (t < ntile) {
              mbar_wait<5>(smem_u32(&ctrl->q_full[t]), (q_ph >> t) & 1);
              q_ph ^= 1u << t;
            }
          // S_t(sub) = Q_t K[sub]^T into S buffer sub & 1; k_lo = descriptor word of the K tile
          auto issue_qk = [&](int t, int sub, uint32_t k_lo) {
            const uint32_t kk = k_lo + (((sub % kNB) * (kSubN * 128)) >> 4);
            const uint32_t qt_lo = q_lo + ((t * Cfg::kTileBytes) >> 4);
            const uint32_t ts = tmem_base + t * 128 + (sub % kNB) * kSubN;
#pragma unroll
            for (int k = 0; k < D / 16; ++k) {
              const uint32_t off = ((k >> 2) * Cfg::kBoxBytes + (k & 3) * 32) >> 4;
              umma_ss(ts, mk_desc(qt_lo + off), mk_desc(kk + off), Cfg::kIdescQK, k > 0);
            }
            umma_commit(bar_s + (2 * t + (sub % kNB)) * 8);
            if (sub == nsub - 1) umma_commit(smem_u32(&ctrl->q_empty[t]));   // Q_t may be refilled
          };
          // prologue: S(0), S(1) from K tile 0
          {
            const uint32_t slot = kv_pos % Cfg::kStages;
            mbar_wait<6>(smem_u32(&ctrl->kv_full[slot]), (kv_pos / Cfg::kStages) & 1);
            tc_fence_after();
            const uint32_t k_lo = kv_lo + kLoKmajor + ((slot * Cfg::kTileBytes) >> 4);
            for (int sub = 0; sub < kNB && sub < nsub; ++sub)
#pragma unroll
              for (int t = 0; t < 2; ++t)
                if (t < ntile) issue_qk(t, sub, k_lo);
            umma_commit(smem_u32(&ctrl->kv_empty[slot]));   // K tile 0: both sub-tiles issued
          }
          uint32_t vslot = 0, kslot = 0;
          for (int sub = 0; sub < nsub; ++sub) {
            const int bufi = sub % kNB;
            if (bufi == 0) {
              const uint32_t vpos = kv_pos + 2 * (sub / kNB) + 1;   // V tile sub / kNB
              vslot = vpos % Cfg::kStages;
              mbar_wait<7>(smem_u32(&ctrl->kv_full[vslot]), (vpos / Cfg::kStages) & 1);
            }
            const int nxt = sub + kNB;                   // S sub-tile issued behind this PV
            const bool has_next = nxt < nsub;
            const int ksteps = (min(kSubN, n_keys - sub * kSubN) + 15) >> 4;
            const uint32_t v_lo =
                kv_lo + kLoMNmajor + ((vslot * Cfg::kTileBytes + bufi * (kSubN * 128)) >> 4);
#pragma unroll
            for (int t = 0; t < 2; ++t) {
              if (t < ntile) {
                if (sub == 0) {
                  // the epilogue group must have drained O_t of the previous item
                  mbar_wait<8>(smem_u32(&ctrl->o_empty[t]), ((od_ph >> t) & 1) ^ 1);
                  od_ph ^= 1u << t;
                }
                mbar_wait<9>(bar_p + (2 * t + bufi) * 8, (pf_ph >> (2 * t + bufi)) & 1);
                pf_ph ^= 1u << (2 * t + bufi);
                tc_fence_after();
                const uint32_t tp = tmem_base + t * 128 + bufi * kSubN;
                const uint32_t to = tmem_base + 256 + t * D;
#pragma unroll
                for (int k = 0; k < kSubN / 16; ++k) {
                  // A = P_t[:, 16k..16k+16) : 8 TMEM columns of packed bf16 pairs
                  // B = V rows [16k, 16k+16) of the sub-tile: MN-major, 8-row groups 1024 B
                  //     apart, the two 64-column halves (D = 128) one box apart
                  if (k < ksteps)
                    umma_ts(to, tp + k * 8, mk_desc(v_lo + k * (2048 >> 4)), Cfg::kIdescPV,
                            (sub > 0 || k > 0) ? 1u : 0u);
                }
                umma_commit(smem_u32(&ctrl->pv_done[t]));
                if (has_next) {
                  if (t == 0 && (nxt % kNB) == 0) {
                    const uint32_t kpos = kv_pos + 2 * (nxt / kNB);   // K tile nxt / kNB
                    kslot = kpos % Cfg::kStages;
                    mbar_wait<10>(smem_u32(&ctrl->kv_full[kslot]), (kpos / Cfg::kStages) & 1);
                    tc_fence_after();
                  }
                  issue_qk(t, nxt, kv_lo + kLoKmajor + ((kslot * Cfg::kTileBytes) >> 4));
                } else if (sub == nsub - 1) {
                  umma_commit(smem_u32(&ctrl->o_full[t]));
                }
              }
            }
            // V tile done after its last sub-tile; K tile done after its last S sub-tile
            if (bufi == kNB - 1 || sub == nsub - 1) umma_commit(smem_u32(&ctrl->kv_empty[vslot]));
            if (has_next && ((nxt % kNB) == kNB - 1 || nxt == nsub - 1))
              umma_commit(smem_u32(&ctrl->kv_empty[kslot]));
          }
          kv_pos += 2 * nt;
        }
        mbar_arrive(smem_u32(&ctrl->item_empty[islot]));
      }
    }
    __syncwarp();
  } else if (warp == kConvWarp0 || warp == kConvWarp0 + 1) {
    // ================================================================= converters
    setmaxnreg_dec<kOtherRegs>();
    if constexpr (kConvert) {
      const int ctid = threadIdx.x - kConvWarp0 * 32;  // 0..63
      uint32_t kv_it = 0, raw_it = 0;
      for (uint32_t n = 0;; ++n) {
        const int islot = n & 1;
        mbar_wait<11>(smem_u32(&ctrl->item_full[islot]), (n >> 1) & 1);
        const WorkItem it = ctrl->items[islot];
        if (!it.valid) break;
        const int nt = (it.n_keys + kTileN - 1) / kTileN;
        for (int jj = 0; jj < 2 * nt; ++jj) {  // K0 V0 K1 V1 ...
          const uint32_t slot = kv_it % Cfg::kStages, ph = (kv_it / Cfg::kStages) & 1;
          mbar_wait<12>(smem_u32(&ctrl->kv_empty[slot]), ph ^ 1);
          const uint32_t tile = kv_smem + slot * Cfg::kTileBytes;
#pragma unroll 1
          for (int c = 0; c < Cfg::kRawPerTile; ++c) {
            const uint32_t rslot = raw_it % Cfg::kRawStages, rph = (raw_it / Cfg::kRawStages) & 1;
            mbar_wait<13>(smem_u32(&ctrl->raw_full[rslot]), rph);
            const uint32_t raw = raw_smem + rslot * Cfg::kRawSlotBytes;
            if constexpr (KV == KV_FP8) {
              constexpr int PPR = D / 16;                   // 16-byte pieces per row
              constexpr int NP = Cfg::kRawRows * PPR;
#pragma unroll 4
              for (int p = ctid; p < NP; p += kConvThreads) {
                const int row = p / PPR, c16 = p % PPR;
                const uint4 v = lds128(raw + p * 16);
                uint32_t o[8];
                e4m3x4_to_f16x4(v.x, o[0], o[1]);
                e4m3x4_to_f16x4(v.y, o[2], o[3]);
                e4m3x4_to_f16x4(v.z, o[4], o[5]);
                e4m3x4_to_f16x4(v.w, o[6], o[7]);
                const int ca = 2 * c16, cb = 2 * c16 + 1;
                const uint32_t rbase = tile + row * 128;
                sts128(rbase + (ca >> 3) * Cfg::kBoxBytes + (((ca & 7) ^ (row & 7)) << 4), o[0], o[1],
                       o[2], o[3]);
                sts128(rbase + (cb >> 3) * Cfg::kBoxBytes + (((cb & 7) ^ (row & 7)) << 4), o[4], o[5],
                       o[6], o[7]);
              }
            } else {
              constexpr int PPR = D / 8;                    // 32-byte pieces (8 floats) per row
              constexpr int NP = Cfg::kRawRows * PPR;
#pragma unroll 2
              for (int p = ctid; p < NP; p += kConvThreads) {
                const int row = c * Cfg::kRawRows + p / PPR, cc = p % PPR;
                const uint4 a = lds128(raw + p * 32), b = lds128(raw + p * 32 + 16);
                const uint32_t o0 = pack_bf16x2(__uint_as_float(a.x), __uint_as_float(a.y));
                const uint32_t o1 = pack_bf16x2(__uint_as_float(a.z), __uint_as_float(a.w));
                const uint32_t o2 = pack_bf16x2(__uint_as_float(b.x), __uint_as_float(b.y));
                const uint32_t o3 = pack_bf16x2(__uint_as_float(b.z), __uint_as_float(b.w));
                sts128(tile + row * 128 + (cc >> 3) * Cfg::kBoxBytes + (((cc & 7) ^ (row & 7)) << 4),
                       o0, o1, o2, o3);
              }
            }
            mbar_arrive(smem_u32(&ctrl->raw_empty[rslot]));
            ++raw_it;
          }
          fence_proxy_async_smem();   // generic-proxy tile writes -> visible to tcgen05.mma
          mbar_arrive(smem_u32(&ctrl->kv_full[slot]));
          ++kv_it;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->item_empty[islot]));
      }
    }
  } else if (warp < 8) {
    // ================================================================= softmax groups
    setmaxnreg_inc<kSoftmaxRegs>();
    const int t = warp >> 2;                 // candidate tile of this group
    const int tid128 = threadIdx.x & 127;    // row within the tile == TMEM lane
    const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tm_s = tmem_base + lane_base + t * 128;
    const uint32_t tm_o = tmem_base + lane_base + 256 + t * D;
    const uint32_t q_tile_smem = q_smem + t * Cfg::kTileBytes;
    uint32_t sf_it[2] = {0, 0};              // s_full phase counters per S buffer
    uint32_t pv_cnt = 0;                     // PV sub-tile MMAs of this tile issued so far (all items)
    // share of exponentials on the FMA pipe: -1 none, 1 -> 25 %, 0 -> 50 %.  Measured (A/B in one
    // run): d = 64 bf16 cache +7.5 % at 25 %, +3.6 % at 50 %; d = 128 -2.5 %; FP8 cache -7 % with the bf16
    // converters, -0.6 % / -3.7 % at 25 % / 50 % with the fp16 route -- so only d = 64 with a bf16 cache uses it.
    constexpr int kPolyMask = (D == 64 && KV == KV_BF16) ? 1 : -1;
    const bool has_self = (args.k_self != nullptr);
    const bool q32 = args.q_is_f32 != 0;
    const size_t row_stride = static_cast<size_t>(args.H) * D;
    bool q_prefetched = false;

    // element offset of row 0 of this group's tile of an item, and its valid row count
    auto tile_elem0_of = [&](const WorkItem& w) -> size_t {
      return ((static_cast<size_t>(w.layer) * w.total_q + w.q_row0 + t * kTileM) * args.H + w.h) * D;
    };
    auto issue_q = [&](const WorkItem& w) {
      const int rows = min(kTileM, w.n_rows - t * kTileM);
      if (q32 || Cfg::kF16)
        load_q_tile<D, Cfg::kF16>(q_tile_smem, args.q, q32, tile_elem0_of(w), row_stride, rows, tid128);
      else
        load_q_tile_async<D>(q_tile_smem, args.q, tile_elem0_of(w), row_stride, rows, tid128);
    };

    for (uint32_t n = 0;; ++n) {
      const int islot = n & 1;
      mbar_wait<14>(smem_u32(&ctrl->item_full[islot]), (n >> 1) & 1);
      const WorkItem it = ctrl->items[islot];
      if (!it.valid) break;
      const int rows_here = min(kTileM, it.n_rows - t * kTileM);  // <= 0: tile inactive
      const int nsub = (rows_here > 0) ? (it.n_keys + kSubN - 1) / kSubN : 0;
      // Prefetch the NEXT item's Q tile as soon as this item's last S_t MMA has read Q_t.
      auto prefetch_next_q = [&]() {
        // (the wait stays even when the producer loads Q by TMA: a group must not release item n
        // before item n+1 is published -- without it, CTAs with key-less items in between hung)
        const uint32_t n1 = n + 1;
        mbar_wait<15>(smem_u32(&ctrl->item_full[n1 & 1]), (n1 >> 1) & 1);
        if (q_by_tma) return;
        const WorkItem nx = ctrl->items[n1 & 1];
        if (nx.valid && nx.n_rows > t * kTileM && nx.n_keys > 0) {
          issue_q(nx);
          q_prefetched = true;
        }
      };
      if (rows_here > 0) {
        const bool row_valid = tid128 < rows_here;
        const size_t my_elem0 = tile_elem0_of(it) + static_cast<size_t>(tid128) * row_stride;
        if (nsub > 0 && !q_by_tma) {
          if (!q_prefetched) issue_q(it);
          cp_async_wait_all();
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl->q_full[t]));
          q_prefetched = false;
        }
        const int sidx = args.scale_per_user ? (it.layer * args.B + it.b) * args.H + it.h : it.layer * args.H + it.h;
        const float ks = args.k_scale ? __ldg(args.k_scale + sidx) : 1.0f;
        const float c_log2 = args.scale_log2 * ks;  // multiplies raw S

        // running state, log2 units. The self key (first split only) seeds it.
        const bool self_here = has_self && it.split == 0;
        float m_used = -INFINITY, l = 0.f, s_self = 0.f;
        if (self_here) {
          s_self = row_valid ? row_dot<D>(args.q, args.k_self, q32, my_elem0) * args.scale_log2
                             : 0.f;
          m_used = s_self;
          l = 1.f;
        }

        // exp-phase ping-pong between the two groups (both tiles active): a warp's step is a
        // latency-bound part (barrier, TMEM load, row max) and a MUFU-bound part (64 ex2 at
        // 8 cycles each per SMSP).  The two softmax warps of an SMSP drift into lockstep
        // unless forced apart, and then nothing hides either part; handing the MUFU phase
        // back and forth keeps them in anti-phase.  Barrier 1 = "group 0 may go", 2 = "group 1".
        const bool pingpong = (it.n_rows > kTileM) && nsub > 0;
        if (pingpong && t == 1) named_bar_arrive(1, 256);

        // One 64-key step.  The last step of an item (tail masking, next Q prefetch) is a separate
        // instantiation so that the steady-state loop body stays as small as possible: the kernel
        // is sensitive to the instruction footprint of this loop.
        auto step = [&](const int sub, auto last_tag) {
          constexpr bool kLast = decltype(last_tag)::value;
          const int bufi = sub % kNB;
          const uint32_t tm_sb = tm_s + bufi * kSubN;
          mbar_wait<16>(smem_u32(&ctrl->s_full[t][bufi]), sf_it[bufi] & 1);
          ++sf_it[bufi];
          tc_fence_after();
          if (kLast) prefetch_next_q();   // every S_t MMA of this item is complete
          uint32_t sr[kSubN];
#pragma unroll
          for (int c0 = 0; c0 < kSubN; c0 += 32) tmem_ld32(tm_sb + c0, &sr[c0]);
          tmem_wait_ld_regs(sr);
          const int keys_here = it.n_keys - sub * kSubN;  // may exceed 64
          if (kLast && keys_here < kSubN) {
#pragma unroll
            for (int c = 0; c < kSubN; ++c)
              if (c >= keys_here) sr[c] = 0xff800000u;  // -inf
          }
          // row max: 4 independent chains
          float mx0 = __uint_as_float(sr[0]), mx1 = __uint_as_float(sr[1]);
          float mx2 = __uint_as_float(sr[2]), mx3 = __uint_as_float(sr[3]);
#pragma unroll
          for (int c = 4; c < kSubN; c += 4) {
            mx0 = fmaxf(mx0, __uint_as_float(sr[c + 0]));
            mx1 = fmaxf(mx1, __uint_as_float(sr[c + 1]));
            mx2 = fmaxf(mx2, __uint_as_float(sr[c + 2]));
            mx3 = fmaxf(mx3, __uint_as_float(sr[c + 3]));
          }
          const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
          const float m_new = fmaxf(m_used, mx * c_log2);
          const bool need = m_new > m_used + kRescaleTau;
          if (sub == 0) {
            // nothing accumulated in O yet (first PV overwrites); only l may hold the self weight
            if (need) {
              l *= ex2_approx(m_used - m_new);
              m_used = m_new;
            }
          } else if (__any_sync(0xffffffffu, need)) {
            // PV(sub-1) may still be accumulating into O_t: wait for it before touching O
            mbar_wait<17>(smem_u32(&ctrl->pv_done[t]), (pv_cnt - 1) & 1);
            tc_fence_after();
            const float alpha = need ? ex2_approx(m_used - m_new) : 1.0f;
#pragma unroll
            for (int c0 = 0; c0 < D; c0 += 16) {
              uint32_t orr[16];
              tmem_ld16(tm_o + c0, orr);
              tmem_wait_ld_regs(orr);
#pragma unroll
              for (int c = 0; c < 16; ++c)
                orr[c] = __float_as_uint(__uint_as_float(orr[c]) * alpha);
              tmem_st16(tm_o + c0, orr);
            }
            l *= alpha;
            if (need) m_used = m_new;
          }
          // P = exp2(S*c - m) as bf16 pairs for the PV MMA, written back over S in chunks of
          // 32 keys.  The row sum (4 chains) adds the bf16-ROUNDED weights, i.e. exactly
          // what the MMA multiplies, so out = sum(p~ v) / sum(p~) stays a convex combination
          // of V rows (matters when few keys dominate).
          if (pingpong) named_bar_sync(1 + t, 256);
          float2 sumA = make_float2(0.f, 0.f), sumB = make_float2(0.f, 0.f);
          const float2 c2 = make_float2(c_log2, c_log2), nm2 = make_float2(-m_used, -m_used);
#pragma unroll
          for (int c0 = 0; c0 < kSubN; c0 += 32) {
            uint32_t pr[16];
#pragma unroll
            for (int c = 0; c < 32; c += 4) {
              const float2 x01 = ffma2(make_float2(__uint_as_float(sr[c0 + c + 0]),
                                                   __uint_as_float(sr[c0 + c + 1])), c2, nm2);
              const float2 x23 = ffma2(make_float2(__uint_as_float(sr[c0 + c + 2]),
                                                   __uint_as_float(sr[c0 + c + 3])), c2, nm2);
              const float p0 = ex2_approx(x01.x), p1 = ex2_approx(x01.y);
              float p2, p3;
              // d = 64: one ex2 per 256 tensor FLOPs makes MUFU (16 / clk / SM) the ceiling, so
              // a share of the exponentials is evaluated as a polynomial on the FMA pipe
              if (kPolyMask >= 0 && ((c >> 2) & kPolyMask) == 0) {
                const float2 e = ex2_poly2(x23);
                p2 = e.x;
                p3 = e.y;
              } else {
                p2 = ex2_approx(x23.x);
                p3 = ex2_approx(x23.y);
              }
              const uint32_t w01 = Cfg::kF16 ? pack_f16x2(p0, p1) : pack_bf16x2(p0, p1);
              const uint32_t w23 = Cfg::kF16 ? pack_f16x2(p2, p3) : pack_bf16x2(p2, p3);
              pr[(c >> 1) + 0] = w01;
              pr[(c >> 1) + 1] = w23;
              if (Cfg::kF16) {
                add_f16x2_f32(sumA.x, sumA.y, w01);
                add_f16x2_f32(sumB.x, sumB.y, w23);
              } else {
                add_bf16x2_f32(sumA.x, sumA.y, w01);
                add_bf16x2_f32(sumB.x, sumB.y, w23);
              }
            }
            tmem_st16(tm_sb + (c0 >> 1), pr);
          }
          if (pingpong && !(t == 1 && kLast)) named_bar_arrive(2 - t, 256);
          l += (sumA.x + sumA.y) + (sumB.x + sumB.y);
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl->p_full[t][bufi]));
          ++pv_cnt;
        };
        for (int sub = 0; sub + 1 < nsub; ++sub) step(sub, cuda::std::false_type{});
        if (nsub > 0) step(nsub - 1, cuda::std::true_type{});
        if (nsub == 0) prefetch_next_q();

        // ---------------------------------------------------------- hand over to the epilogue
        const bool partial = args.num_splits > 1;
        ctrl->epi_inv[islot][t][tid128] = partial ? 1.0f : (l > 0.f ? 1.0f / l : 0.f);
        ctrl->epi_wself[islot][t][tid128] = self_here ? ex2_approx(s_self - m_used) : 0.f;
        if (partial && row_valid) {
          const size_t prow =
              ((static_cast<size_t>(it.layer) * it.total_q + it.q_row0 + t * kTileM + tid128) *
                   args.H + it.h) * args.num_splits + it.split;
          args.part_ml[prow * 2 + 0] = m_used;
          args.part_ml[prow * 2 + 1] = l;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->l_ready[t]));
      } else {
        // inactive tile: its Q buffer is idle, so the next item's tile can be staged now
        prefetch_next_q();
      }
      mbar_arrive(smem_u32(&ctrl->item_empty[islot]));
    }
  } else {
    // ================================================================= epilogue group (a7)
    setmaxnreg_dec<kEpilogueRegs>();
    const int ew = warp - kEpiWarp0;                     // TMEM lane quarter of this warp
    const uint32_t lane_base = static_cast<uint32_t>(ew * 32) << 16;
    const uint32_t stage = epi_smem + ew * Cfg::kEpiWarpBytes;
    const bool has_self = (args.v_self != nullptr);
    const bool q32 = args.q_is_f32 != 0;
    const bool partial = args.num_splits > 1;
    uint32_t lr_it[2] = {0, 0}, of_it[2] = {0, 0};
    for (uint32_t n = 0;; ++n) {
      const int islot = n & 1;
      mbar_wait<18>(smem_u32(&ctrl->item_full[islot]), (n >> 1) & 1);
      const WorkItem it = ctrl->items[islot];
      if (!it.valid) break;
      const int nt = (it.n_keys + kTileN - 1) / kTileN;
      const bool self_here = has_self && it.split == 0;
      const float vs = args.v_scale ? __ldg(args.v_scale + (args.scale_per_user ? (it.layer * args.B + it.b) * args.H + it.h
                                                                                 : it.layer * args.H + it.h))
                                    : 1.0f;
#pragma unroll 1
      for (int t = 0; t < 2; ++t) {
        const int rows_here = min(kTileM, it.n_rows - t * kTileM);
        if (rows_here <= 0) break;
        mbar_wait<19>(smem_u32(&ctrl->l_ready[t]), lr_it[t] & 1);
        ++lr_it[t];
        if (nt > 0) {
          mbar_wait<20>(smem_u32(&ctrl->o_full[t]), of_it[t] & 1);
          ++of_it[t];
          tc_fence_after();
        }
        const int row = ew * 32 + lane;                  // row of this thread within the tile
        const float inv = ctrl->epi_inv[islot][t][row];
        const float sc = vs * inv;                                     // out = O * sc + ws * v_self
        const float ws = ctrl->epi_wself[islot][t][row] * inv;
        const size_t grow0 = static_cast<size_t>(it.layer) * it.total_q + it.q_row0 + t * kTileM;
        // candidate-side element offset of (row 0 of the tile, head h)
        const size_t q_elem0 = (grow0 * args.H + it.h) * D;
        float* dst0;
        size_t dst_stride;
        if (!partial) {
          dst0 = args.out + q_elem0;
          dst_stride = static_cast<size_t>(args.H) * D;
        } else {
          dst0 = args.part_o + ((grow0 * args.H + it.h) * args.num_splits + it.split) * D;
          dst_stride = static_cast<size_t>(args.H) * args.num_splits * D;
        }
        // transposed read-back: 8 lanes cover one row's 128-byte line, 4 rows per access
        const int rr = lane >> 3, cq = lane & 7;
        float* gp = dst0 + static_cast<size_t>(ew * 32 + rr) * dst_stride + cq * 4;
        const size_t gstep = 4 * dst_stride;
        const int rem = rows_here - (ew * 32 + rr);      // row 4k + rr of this warp valid iff 4k < rem
        const uint32_t st_w = stage + lane * kEpiRowBytes;
        const uint32_t st_r = stage + rr * kEpiRowBytes + cq * 16;
        const bool add_self = self_here && row < rows_here;
        const size_t se0 = q_elem0 + static_cast<size_t>(row) * args.H * D;
        const uint32_t tm_o = tmem_base + lane_base + 256 + t * D;
        const float2 sc2 = make_float2(sc, sc);
        if (args.out_tma && !partial && !self_here && nt > 0 && rows_here == kTileM) {
          // full tile, plain output: each 32 x 32 block is staged as a dense 128-byte-swizzled box
          // and leaves through one TMA store; the warp only waits until the engine has READ the
          // box before refilling it, never for the write to land
          const int grow = static_cast<int>(grow0) + ew * 32;
          const uint32_t sw_row = stage + lane * 128;
          uint32_t orr[32];
          tmem_ld32(tm_o, orr);
#pragma unroll 1
          for (int c0 = 0; c0 < D; c0 += 32) {
            tmem_wait_ld_regs(orr);
            if (c0 + 32 == D) {
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive(smem_u32(&ctrl->o_empty[t]));
            }
            if (lane == 0) bulk_wait_read_all();
            __syncwarp();
#pragma unroll
            for (int c = 0; c < 32; c += 4) {
              const float2 a = fmul2(make_float2(__uint_as_float(orr[c]), __uint_as_float(orr[c + 1])), sc2);
              const float2 b2 = fmul2(make_float2(__uint_as_float(orr[c + 2]), __uint_as_float(orr[c + 3])), sc2);
              sts128(sw_row + (((c >> 2) ^ (lane & 7)) << 4), __float_as_uint(a.x), __float_as_uint(a.y),
                     __float_as_uint(b2.x), __float_as_uint(b2.y));
            }
            if (c0 + 32 < D) tmem_ld32(tm_o + c0 + 32, orr);   // next block: overlaps the store hand-off
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&tmap_out, stage, it.h * D + c0, grow);
              bulk_commit();
            }
          }
        } else {
        if (lane == 0) bulk_wait_read_all();   // a TMA store of an earlier tile may still read the block
        __syncwarp();
#pragma unroll 1
        for (int c0 = 0; c0 < D; c0 += 32) {
          uint32_t orr[32];
          if (nt > 0) {
            tmem_ld32(tm_o + c0, orr);
            tmem_wait_ld_regs(orr);
            if (c0 + 32 == D) {
              // the accumulator is in registers: hand O_t back before staging / storing the
              // last block, so the next item's first PV waits one block less
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive(smem_u32(&ctrl->o_empty[t]));
            }
          } else {
#pragma unroll
            for (int c = 0; c < 32; ++c) orr[c] = 0u;
          }
          if (!self_here) {
#pragma unroll
            for (int c = 0; c < 32; c += 4) {
              const float2 a = fmul2(make_float2(__uint_as_float(orr[c]), __uint_as_float(orr[c + 1])), sc2);
              const float2 b2 = fmul2(make_float2(__uint_as_float(orr[c + 2]), __uint_as_float(orr[c + 3])), sc2);
              sts128(st_w + c * 4, __float_as_uint(a.x), __float_as_uint(a.y), __float_as_uint(b2.x),
                     __float_as_uint(b2.y));
            }
          } else {
#pragma unroll
            for (int c = 0; c < 32; c += 8) {
              float sv[8];
#pragma unroll
              for (int k = 0; k < 8; ++k) sv[k] = 0.f;
              if (add_self) {
                if (!q32) {
                  const uint4 x = __ldg(reinterpret_cast<const uint4*>(
                      static_cast<const __nv_bfloat16*>(args.v_self) + se0 + c0 + c));
                  const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                  for (int k = 0; k < 4; ++k) {
                    sv[2 * k + 0] = __uint_as_float(w[k] << 16);
                    sv[2 * k + 1] = __uint_as_float(w[k] & 0xffff0000u);
                  }
                } else {
                  const float4* s4 = reinterpret_cast<const float4*>(
                      static_cast<const float*>(args.v_self) + se0 + c0 + c);
                  const float4 a = __ldg(s4), b4 = __ldg(s4 + 1);
                  sv[0] = a.x; sv[1] = a.y; sv[2] = a.z; sv[3] = a.w;
                  sv[4] = b4.x; sv[5] = b4.y; sv[6] = b4.z; sv[7] = b4.w;
                }
              }
              float o[8];
#pragma unroll
              for (int k = 0; k < 8; ++k) o[k] = fmaf(ws, sv[k], __uint_as_float(orr[c + k]) * sc);
              sts128(st_w + c * 4, __float_as_uint(o[0]), __float_as_uint(o[1]), __float_as_uint(o[2]),
                     __float_as_uint(o[3]));
              sts128(st_w + c * 4 + 16, __float_as_uint(o[4]), __float_as_uint(o[5]),
                     __float_as_uint(o[6]), __float_as_uint(o[7]));
            }
          }
          __syncwarp();
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const uint4 v = lds128(st_r + k * (4 * kEpiRowBytes));
            if (4 * k < rem) stg128_stream(gp + k * gstep + c0, v);
          }
          __syncwarp();
        }
        }

      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->item_empty[islot]));
    }
    if (lane == 0) bulk_wait_all();   // outstanding TMA stores must land before the CTA retires
  }

  // ------------------------------------------------------------------ teardown
  if (diag) {
    unsigned long long t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
    unsigned long long* dst = reinterpret_cast<unsigned long long*>(args.counter + 16);
    dst[0] = static_cast<unsigned long long>(clock64()) - diag_c0;
    dst[1] = t1 - diag_t0;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kMmaWarp) {
    tc_fence_after();
    tmem_dealloc(tmem_base, kTmemCols);
  }
}

}  // namespace upr
