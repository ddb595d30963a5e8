// attn2_kernel.cuh -- ranking-head cross-attention forward on a CTA PAIR (steps a2-a7 of
// SURVEY.md 8(a)) for bf16 K/V, d = 128: the kernel the tensor-bound configs run on.
//
// Same mathematics as attn_kernel.cuh (out = softmax(scale * q K^T) V per candidate over its
// user's cached history; optional self key/value), different mapping:
//
//  * the self term (a6) is ONE MORE KEY TILE per 128-row Q tile: the candidates' own keys / values, loaded by TMA
//    in the Q tile's row order, under the identity mask of PAPER.md:198 (row r sees key r only).  It goes through
//    the same S MMA, softmax step and PV MMA as a history tile, so there is no per-item side path (the per-row dot
//    products and value rows read from global memory cost ~10 000 cycles per item when they were one).
//
//  * a cluster of two CTAs (two SMs) owns a work item = (layer, user, KV head, history split,
//    block of <= 256 query rows); each CTA holds ONE 128-row Q tile and its 128 lanes of TMEM;
//    tcgen05.mma.cta_group::2 (M = 256) is issued by one thread of the pair's leader and runs on
//    both SMs.  The B operand is split between the two CTAs' shared memories: for S = Q K^T each
//    CTA streams HALF of every 128-key K tile (64 keys), for O += P V each CTA streams half of V's
//    d columns -- every K/V byte enters the pair once, and per-CTA operand traffic halves.
//  * S tiles are 128 keys wide (N = 128: the Q operand is re-read half as often as with the
//    64-key sub-tiles of the 1-CTA kernel), two S buffers per CTA.
//  * O is DOUBLE-BUFFERED (2 x 128 columns): the epilogue drains item n while the MMAs of item
//    n+1 accumulate into the other buffer; S and PV issue run as one stream of key tiles across
//    item boundaries (the S tile two ahead is issued behind each PV), so an item boundary costs
//    no drain and no pipeline refill.
//  * the two softmax warpgroups of a CTA work on the SAME 128 rows, two threads per row: group wg takes
//    columns [64 wg, +64) of every key tile.  The half tiles form one sequence of online-softmax steps;
//    a step reads the reference maximum its predecessor published (named barriers between the two warps
//    of a lane quarter), applies the lazy-rescale rule and publishes -- no symmetric exchange.
//  * grouped queries (H_kv < H_q, "KV heads"): the G = H_q / H_kv query heads that
//    share a KV head are folded into M -- a tile holds 128/G candidates x G heads (g-major) --
//    so a K/V tile is reused G times more often.
//  * K/V come through one 2-D tensor map over [rows, d]: the packed decode cache, or the paper's
//    pool [L, S, H_kv, n, D] read in place through slot_ids (zero copy).
//  * work items are handed out longest-first from the tables upr_schedule_kernel builds.
//
// Roles per CTA (512 threads): warps 0-3 / 4-7 softmax groups, 8 producer (+ scheduler; the
// leader's fetches the item index and forwards it to the peer), 9 MMA issuer (leader only), 10-11
// spare, 12-15 epilogue.  TMEM: S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <cuda/std/type_traits>

#include "ptx.cuh"

namespace upr {
namespace pair {

constexpr int kD = 128;
constexpr int kThreads = 512;
constexpr int kRows = 128;            // query rows per CTA == TMEM lanes
constexpr int kKeys = 128;            // keys per tile
constexpr int kItemSlots = 4;
constexpr int kKvSlots = 8;           // ring of half tiles: K0 V0 K1 V1 ...
constexpr int kHalfBytes = 16384;     // K half: 64 keys x 128 d; V half: 128 keys x 64 d (bf16)
constexpr int kKBoxBytes = 64 * 128;  // one [64 keys x 64 d] box of the K half
constexpr int kQBoxBytes = kRows * 128;   // one [128 rows x 64 d] box of the Q tile
constexpr int kQBytes = 2 * kQBoxBytes;
constexpr int kEpiWarpBytes = 5120;   // 32 x 144 B rounded up to 1024 (see attn_kernel.cuh)
constexpr int kEpiRowBytes = 144;
constexpr int kSoftmaxRegs = 168;
constexpr int kOtherRegs = 56;
constexpr int kEpilogueRegs = 88;
static_assert(256 * kSoftmaxRegs + 128 * kOtherRegs + 128 * kEpilogueRegs <= kThreads * 128,
              "setmaxnreg budgets exceed the CTA's register allocation");
constexpr int kProducerWarp = 8, kMmaWarp = 9, kHelpWarp0 = 10, kEpiWarp0 = 12;
constexpr float kTau = 8.0f;          // lazy-rescale threshold, log2 units
// named barriers of the reference-maximum hand-over between the two softmax groups, one pair per TMEM lane quarter q
// (64 threads each: the two warps that share rows [32 q, +32)): group 0 publishes on kBarAB + q, group 1 on kBarBA + q
constexpr int kBarAB = 1, kBarBA = 5;

struct Args {
  const void* q;          // bf16 [n_layers, total_q, H_q, 128]
  const void* k_self;
  const void* v_self;
  float* out;             // fp32, same shape
  const int32_t* seq_lens;
  const int32_t* cand_offsets;
  const int32_t* slot_ids;   // pool mode, else nullptr
  const int32_t* iprefix;    // tables of upr_schedule_kernel
  const int32_t* order;
  const int32_t* rowoff;
  unsigned int* counter;
  float* part_o;          // split-K partials [n_layers][total_q][H_q][ns][128]
  float* part_ml;         //                  [n_layers][total_q][H_q][ns][2]
  int B, H_q, H_kv, G, cpt;  // cpt = 128 / G candidates per tile
  int n_layers, num_splits;
  int pool_S, pool_n;
  int total_q;
  int out_tma;
  int causal;             // candidate c of user b (local index cl) sees keys j <= cl + (L_b - C_b): history prefill
  float scale_log2;
};

struct Item {
  int valid;
  int layer, hkv, split;
  int c0;        // first candidate (global index) of the block
  int cands;     // candidates in the block, 1 .. 2 * cpt
  int kv_row0;   // row of the split's first key in the [rows, d] view of K / V
  int n_keys;    // keys of the split's range (>= 0)
  int n_self;    // self tiles appended behind the history tiles: 0, or one per 128-row Q tile with candidates
  int lim0;      // causal mode: keys visible to the block's first candidate (row r of the block sees lim0 + r);
                 // otherwise 1 << 30
};

struct __align__(16) Ctrl {
  uint64_t item_full[kItemSlots], item_empty[kItemSlots];
  uint64_t idx_full[kItemSlots];   // peer: the leader's item index has landed in idx_ring
  uint64_t idx_free[kItemSlots];   // leader: the peer has read idx_ring[slot] (remote arrive)
  uint64_t kv_full[kKvSlots], kv_empty[kKvSlots];
  uint64_t q_full[2], q_empty[2];
  uint64_t s_full[2];
  uint64_t p_full[2][2];           // [S buffer][half]: leader's copy collects both CTAs' arrivals
  uint64_t pv_done[4];            // PV half-step hs completes phase hs / 4 of pv_done[hs % 4]
  uint64_t o_full[2], o_empty[2];
  uint64_t l_ready[kItemSlots];
  Item items[kItemSlots];
  uint32_t idx_ring[kItemSlots];
  uint32_t tmem_base;
  uint32_t pad_[3];
  int mma_fifo[4][4];                      // MMA thread only: keyed items between its S and PV cursors
  float ref_sh[2][kRows];                  // [publishing group][row]: the row's reference maximum after that group's
                                           // latest half-tile step
  float epi_l[kItemSlots][2][kRows];       // the two groups' partial row sums ...
  float epi_m[kItemSlots][2][kRows];       // ... and the reference maximum each is relative to
};
constexpr int kSmemQ = 2 * kQBytes;                          //  65536
constexpr int kSmemKV = kKvSlots * kHalfBytes;               // 131072
constexpr int kSmemEpi = 4 * kEpiWarpBytes;                  //  20480
constexpr int kSmemCtrl = 11264;
constexpr int kSmemTotal = kSmemQ + kSmemKV + kSmemEpi + kSmemCtrl + 1024;
static_assert(sizeof(Ctrl) <= kSmemCtrl, "control block too large");
static_assert(kSmemTotal <= 232448, "exceeds the 227 KB shared memory of an sm_100 CTA");

__host__ __device__ constexpr uint32_t idesc_pair(int N, int b_mn_major) {
  return make_idesc_bf16(256, N, 0, b_mn_major);
}

// kSelf: the call has a self term (k_self / v_self).  Two instantiations, so that the code of the self tiles costs the
// calls without a self term nothing (registers, scheduling of the steady-state loop).
template <bool kSelf>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
upr_attn_pair_kernel(const __grid_constant__ CUtensorMap tmap_k,    // [rows, 128] bf16, box 64 keys x 64 d
                     const __grid_constant__ CUtensorMap tmap_v,    // [rows, 128] bf16, box 128 keys x 64 d
                     const __grid_constant__ CUtensorMap tmap_q,    // [n_layers*total_q, H_q*128], box cpt x 64
                     const __grid_constant__ CUtensorMap tmap_out,  // fp32 [n_layers*total_q, H_q*128], box 32 x 32
                     const __grid_constant__ CUtensorMap tmap_ks,   // k_self like q, box min(64, cpt) rows x 64
                     const __grid_constant__ CUtensorMap tmap_vs,   // v_self like q, box cpt rows x 64
                     const Args args) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem_aligned = smem_raw + (smem_base - smem_u32(smem_raw));
  const uint32_t q_smem = smem_base;
  const uint32_t kv_smem = q_smem + kSmemQ;
  const uint32_t epi_smem = kv_smem + kSmemKV;
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem_aligned + kSmemQ + kSmemKV + kSmemEpi);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  // rank in the CTA pair (cluster dims (2,1,1): == %cluster_ctarank; written from blockIdx so that the
  // compiler knows it is warp-uniform: 0 = leader; this CTA owns tile `rank` of every item
  const uint32_t rank = blockIdx.x & 1u;
  const bool leader = rank == 0;
  constexpr bool has_self = kSelf;
  const bool partial = args.num_splits > 1;
  const int G = args.G, cpt = args.cpt;

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
    // readers that release an item slot: 8 softmax warps, 4 epilogue warps, the MMA thread (leader only)
    const uint32_t readers = 8 + 4 + (leader ? 1 : 0);
    for (int i = 0; i < kItemSlots; ++i) {
      mbar_init(smem_u32(&ctrl->item_full[i]), 1);
      mbar_init(smem_u32(&ctrl->item_empty[i]), readers);
      mbar_init(smem_u32(&ctrl->idx_full[i]), 1);
      mbar_init(smem_u32(&ctrl->idx_free[i]), 1);
      mbar_init(smem_u32(&ctrl->l_ready[i]), 8);
    }
    for (int i = 0; i < kKvSlots; ++i) {
      mbar_init(smem_u32(&ctrl->kv_full[i]), 1);    // leader's arrive.expect_tx; bytes from both CTAs
      mbar_init(smem_u32(&ctrl->kv_empty[i]), 1);   // multicast commit
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl->q_full[i]), 1);
      mbar_init(smem_u32(&ctrl->q_empty[i]), 1);
      mbar_init(smem_u32(&ctrl->s_full[i]), 1);
      mbar_init(smem_u32(&ctrl->p_full[i][0]), 8);  // 4 softmax warps of a group in each CTA (leader's copy is used)
      mbar_init(smem_u32(&ctrl->p_full[i][1]), 8);
      mbar_init(smem_u32(&ctrl->o_full[i]), 1);
      mbar_init(smem_u32(&ctrl->o_empty[i]), 8);    // 4 epilogue warps of each CTA (leader's copy)
    }
    for (int i = 0; i < 4; ++i) mbar_init(smem_u32(&ctrl->pv_done[i]), 1);
    fence_mbar_init();
  }
  if (warp == kProducerWarp && lane == 0) {
    tma_prefetch_desc(&tmap_k);
    tma_prefetch_desc(&tmap_v);
    tma_prefetch_desc(&tmap_q);
    if (has_self) {
      tma_prefetch_desc(&tmap_ks);
      tma_prefetch_desc(&tmap_vs);
    }
  }
  if (warp == kMmaWarp) {
    tmem_alloc_pair(smem_u32(&ctrl->tmem_base), 512);
    tmem_relinquish_pair();
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();     // both CTAs' barriers are initialised before any remote arrive / TMA signal
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;

  // Valid rows of this CTA's tile of an item: candidates [rank*cpt, rank*cpt + n_here) x G heads
  auto cands_here = [&](const Item& it) { return max(0, min(cpt, it.cands - static_cast<int>(rank) * cpt)); };

  if (warp == kProducerWarp) {
    // ================================================================= scheduler + producer
    setmaxnreg_dec<kOtherRegs>();
    const int W = __ldg(args.iprefix + args.B);               // items per layer
    const long long total_items = static_cast<long long>(W) * args.n_layers;
    const int cpb = 2 * cpt;                                    // candidates per block
    // barriers of the pair's leader, as shared::cluster addresses
    const uint32_t lead_kv_full = mapa_shared(smem_u32(&ctrl->kv_full[0]), 0);
    const uint32_t lead_q_full = mapa_shared(smem_u32(&ctrl->q_full[0]), 0);
    const uint32_t peer_idx_full = mapa_shared(smem_u32(&ctrl->idx_full[0]), 1);
    const uint32_t peer_idx_ring = mapa_shared(smem_u32(&ctrl->idx_ring[0]), 1);
    const uint32_t lead_idx_free = mapa_shared(smem_u32(&ctrl->idx_free[0]), 0);
    uint32_t kv_it = 0;      // ring position of the next half tile
    uint32_t n_keyed = 0;    // items with keys so far (selects the Q buffer)
    for (uint32_t n = 0;; ++n) {
      const int islot = n & (kItemSlots - 1);
      const uint32_t use = n / kItemSlots;
      mbar_wait<1>(smem_u32(&ctrl->item_empty[islot]), (use & 1) ^ 1);
      uint32_t idx = 0;
      if (leader) {
        if (lane == 0) {
          idx = atomicAdd(args.counter, 1u);
          // the peer must have read the previous index held by this ring slot (it may lag behind
          // the leader by any number of key-less items, which need nothing from the pair)
          if (use >= 1) mbar_wait_cluster(smem_u32(&ctrl->idx_free[islot]), (use - 1) & 1);
          st_async_u32(peer_idx_ring + islot * 4, idx, peer_idx_full + islot * 8);
        }
        idx = __shfl_sync(0xffffffffu, idx, 0);
      } else {
        if (lane == 0) mbar_arrive_expect_tx(smem_u32(&ctrl->idx_full[islot]), 4);
        mbar_wait<2>(smem_u32(&ctrl->idx_full[islot]), use & 1);
        idx = ctrl->idx_ring[islot];
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(lead_idx_free + islot * 8);
      }
      if (static_cast<long long>(idx) >= total_items) {
        if (lane == 0) {
          ctrl->items[islot].valid = 0;
          mbar_arrive(smem_u32(&ctrl->item_full[islot]));
        }
        break;
      }
      // ---- decode: position i in the longest-first order with iprefix[i] <= r < iprefix[i+1]
      const int r = static_cast<int>(idx / static_cast<uint32_t>(args.n_layers));
      int lo = 0, hi = args.B;   // invariant: iprefix[lo] <= r < iprefix[hi]
      while (hi - lo > 1) {
        const int step = (hi - lo + 31) / 32;
        const int p = lo + lane * step;
        const int v = (p < hi) ? __ldg(args.iprefix + p) : 0x7fffffff;
        const unsigned le = __ballot_sync(0xffffffffu, v <= r);
        const int c = __popc(le);            // lanes 0..c-1 satisfy (prefix is non-decreasing), c >= 1
        const int nlo = lo + (c - 1) * step;
        hi = min(hi, nlo + step);
        lo = nlo;
      }
      const int p0 = __ldg(args.iprefix + lo);
      const int w_user = __ldg(args.iprefix + lo + 1) - p0;                 // items per layer of this user
      const int local_all = static_cast<int>(idx - static_cast<uint32_t>(args.n_layers) * static_cast<uint32_t>(p0));
      const int layer = local_all / w_user;
      const int local = local_all - layer * w_user;
      const int b = __ldg(args.order + lo);
      const int cb0 = __ldg(args.cand_offsets + b);
      const int Cb = __ldg(args.cand_offsets + b + 1) - cb0;
      const int Lb = __ldg(args.seq_lens + b);
      const int nq = (Cb + cpb - 1) / cpb;
      const int per_h = nq * args.num_splits;
      const int hkv = local / per_h;
      const int rem = local - hkv * per_h;
      const int split = rem / nq;
      const int qblk = rem - split * nq;
      const int nt_user = (Lb + kKeys - 1) / kKeys;
      const int t0 = static_cast<int>((static_cast<long long>(split) * nt_user) / args.num_splits);
      const int t1 = static_cast<int>((static_cast<long long>(split + 1) * nt_user) / args.num_splits);
      const int key0 = t0 * kKeys;
      // causal (prefill, one split): row r of the block sees keys [0, lim0 + r); the block needs the keys its
      // last row sees
      const int lim0 = args.causal ? (Lb - Cb) + qblk * cpb + 1 : (1 << 30);
      const int n_keys = args.causal ? max(0, min(Lb, lim0 + min(cpb, Cb - qblk * cpb) - 1))
                                     : ((t1 > t0) ? (min(Lb, t1 * kKeys) - key0) : 0);
      const int kv_row0 =
          (args.slot_ids != nullptr)
              ? ((layer * args.pool_S + __ldg(args.slot_ids + b)) * args.H_kv + hkv) * args.pool_n + key0
              : (layer * args.H_kv + hkv) * __ldg(args.rowoff + args.B) + __ldg(args.rowoff + b) + key0;
      if (elect_one()) {   // (elect.sync: the compiler then issues the TMA instructions without a per-lane loop)
        Item& it = ctrl->items[islot];
        it.valid = 1;
        it.layer = layer;
        it.hkv = hkv;
        it.split = split;
        it.c0 = cb0 + qblk * cpb;
        it.cands = min(cpb, Cb - qblk * cpb);
        it.kv_row0 = kv_row0;
        it.n_keys = n_keys;
        it.lim0 = lim0;
        // the candidates' own keys (first split only): one tile per 128-row Q tile that holds candidates
        const int n_self = (has_self && split == 0) ? (it.cands > cpt ? 2 : 1) : 0;
        it.n_self = n_self;
        mbar_arrive(smem_u32(&ctrl->item_full[islot]));
        const int nt_hist = (n_keys + kKeys - 1) / kKeys;
        const int nt = nt_hist + n_self;
        if (nt > 0) {
          // ---- this CTA's Q tile: G boxes of cpt candidates x 64 columns per 64-column half
          const int qb = n_keyed & 1;
          if (n_keyed >= 2) mbar_wait<3>(smem_u32(&ctrl->q_empty[qb]), ((n_keyed >> 1) - 1) & 1);
          if (leader) mbar_arrive_expect_tx(smem_u32(&ctrl->q_full[qb]), 2 * kQBytes);
          const int qrow = layer * args.total_q + it.c0 + static_cast<int>(rank) * cpt;
          const uint32_t qdst = q_smem + qb * kQBytes;
          for (int g = 0; g < G; ++g) {
            const int col = (hkv * G + g) * kD;
#pragma unroll
            for (int bx = 0; bx < 2; ++bx)
              tma_load_2d_pair(qdst + bx * kQBoxBytes + g * cpt * 128, &tmap_q, col + bx * 64, qrow,
                               lead_q_full + qb * 8);
          }
          ++n_keyed;
          // ---- K / V half tiles: K_j keys [64*rank, +64) of tile j; V_j columns [64*rank, +64)
          for (int j = 0; j < nt; ++j) {
#pragma unroll
            for (int kv = 0; kv < 2; ++kv) {
              const uint32_t slot = kv_it % kKvSlots;
              const uint32_t ph = (kv_it / kKvSlots) & 1;
              mbar_wait<4>(smem_u32(&ctrl->kv_empty[slot]), ph ^ 1);
              if (leader) mbar_arrive_expect_tx(smem_u32(&ctrl->kv_full[slot]), 2 * kHalfBytes);
              const uint32_t dst = kv_smem + slot * kHalfBytes;
              const uint32_t bar = lead_kv_full + slot * 8;
              if (j >= nt_hist) {
                // self tile t: its 128 keys are the rows of Q tile t (g-major: key g * cpt + cl = candidate cl, head g)
                const int srow0 = layer * args.total_q + it.c0 + (j - nt_hist) * cpt;
                if (kv == 0) {
                  const int kbox = min(64, cpt);      // keys [64 rank, 64 rank + 64) in boxes of kbox rows
                  for (int r0 = static_cast<int>(rank) * 64; r0 < static_cast<int>(rank) * 64 + 64; r0 += kbox) {
                    const int g = r0 / cpt, cl0 = r0 - g * cpt;
                    const uint32_t d2 = dst + (r0 - static_cast<int>(rank) * 64) * 128;
                    tma_load_2d_pair(d2, &tmap_ks, (hkv * G + g) * kD, srow0 + cl0, bar);
                    tma_load_2d_pair(d2 + kKBoxBytes, &tmap_ks, (hkv * G + g) * kD + 64, srow0 + cl0, bar);
                  }
                } else {
                  for (int g = 0; g < G; ++g)       // 128 keys x columns [64 rank, 64 rank + 64)
                    tma_load_2d_pair(dst + g * cpt * 128, &tmap_vs, (hkv * G + g) * kD + static_cast<int>(rank) * 64,
                                     srow0, bar);
                }
              } else if (kv == 0) {
                const int row = kv_row0 + j * kKeys + static_cast<int>(rank) * 64;
                tma_load_2d_pair(dst, &tmap_k, 0, row, bar);
                tma_load_2d_pair(dst + kKBoxBytes, &tmap_k, 64, row, bar);
              } else {
                tma_load_2d_pair(dst, &tmap_v, static_cast<int>(rank) * 64, kv_row0 + j * kKeys, bar);
              }
              ++kv_it;
            }
          }
        }
      }
      __syncwarp();
    }
  } else if (warp == kMmaWarp) {
    // ================================================================= MMA issuer (leader)
    // One stream of key tiles across items.  Per tile g (global count): S(g) = Q K_g^T into S
    // buffer g & 1, later O += P(g) V_g.  S runs up to two tiles ahead of PV, across item
    // boundaries, so the tensor pipe never waits for an item's epilogue or first loads.
    setmaxnreg_dec<kOtherRegs>();
    if (leader) {
    if (elect_one()) {
      constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);   // SBO 1024, version 1, SWIZZLE_128B
      constexpr uint32_t kLoK = (16u >> 4) << 16;                               // K-major operands (Q, K)
      constexpr uint32_t kLoMN = (1024u >> 4) << 16;                            // MN-major V half (one atom wide)
      constexpr uint32_t kIdescS = idesc_pair(kKeys, 0);
      constexpr uint32_t kIdescO = idesc_pair(kD, 1);
      auto mk_desc = [](uint32_t lo) {
        return (static_cast<uint64_t>(kDescHi) << 32) | static_cast<uint64_t>(lo);
      };
      const uint32_t q_lo = ((q_smem & 0x3FFFFu) >> 4) | kLoK;
      const uint32_t kv_lo = (kv_smem & 0x3FFFFu) >> 4;
      // S cursor
      uint32_t s_item = 0;        // next item slot index the S cursor will look at
      int s_nt = 0, s_j = 0;      // tiles of the S cursor's current item / next tile to issue
      uint32_t s_kv = 0;          // ring position of the S cursor's current item's K_0
      uint32_t s_keyed = 0;       // keyed items the S cursor has entered
      bool s_end = false;
      uint32_t gs = 0;            // global tiles S-issued
      // PV cursor: a FIFO (shared memory, private to this thread) of the keyed items between the
      // two cursors; the head entry is cached in registers
      uint32_t f_head = 0, f_tail = 0;   // f_tail - f_head = keyed items entered by S and not finished by PV
      int p_j = 0, p_nkeys = 0, p_slot = 0, p_nt = 0;
      uint32_t p_kv = 0;
      uint32_t gp = 0;            // global tiles PV-issued
      uint32_t p_keyed = 0;       // keyed items the PV cursor has finished
      uint32_t kv_next = 0;       // ring position after the last entered item
      for (;;) {
        // ---- 1. S issue: keep up to two tiles in flight ahead of PV
        while (gs - gp < 2 && !s_end) {
          if (s_j == s_nt) {
            const int islot = s_item & (kItemSlots - 1);
            const uint32_t par = (s_item / kItemSlots) & 1;
            const uint32_t bar = smem_u32(&ctrl->item_full[islot]);
            if (!mbar_test(bar, par)) {
              if (gs != gp) break;      // PV work is pending: never block on the look-ahead
              mbar_wait<5>(bar, par);
            }
            const Item& it = ctrl->items[islot];
            if (!it.valid) {
              s_end = true;
              break;
            }
            const int nt = (it.n_keys + kKeys - 1) / kKeys + it.n_self;
            ++s_item;
            if (nt == 0) {              // key-less item: nothing for the tensor pipe
              mbar_arrive(smem_u32(&ctrl->item_empty[islot]));
              continue;
            }
            s_nt = nt;
            s_j = 0;
            s_kv = kv_next;
            kv_next += 2 * nt;
            const int fi = f_tail & 3;
            ctrl->mma_fifo[fi][0] = it.n_keys;
            ctrl->mma_fifo[fi][1] = islot;
            ctrl->mma_fifo[fi][2] = static_cast<int>(s_kv);
            ctrl->mma_fifo[fi][3] = nt;
            ++f_tail;
            const int qb = s_keyed & 1;
            mbar_wait_cluster(smem_u32(&ctrl->q_full[qb]), (s_keyed >> 1) & 1);
            ++s_keyed;
          }
          const int qb = (s_keyed - 1) & 1;
          const uint32_t kpos = s_kv + 2 * s_j;
          const uint32_t kslot = kpos % kKvSlots;
          mbar_wait_cluster(smem_u32(&ctrl->kv_full[kslot]), (kpos / kKvSlots) & 1);
          tc_fence_after();
          const uint32_t sb = gs & 1;
          const uint32_t a_lo = q_lo + ((qb * kQBytes) >> 4);
          const uint32_t b_lo = kv_lo + kLoK + ((kslot * kHalfBytes) >> 4);
#pragma unroll
          for (int k = 0; k < kD / 16; ++k) {
            const uint32_t a_off = ((k >> 2) * kQBoxBytes + (k & 3) * 32) >> 4;
            const uint32_t b_off = ((k >> 2) * kKBoxBytes + (k & 3) * 32) >> 4;
            umma_ss_pair(tmem_base + sb * kKeys, mk_desc(a_lo + a_off), mk_desc(b_lo + b_off), kIdescS, k > 0);
          }
          umma_commit_pair(smem_u32(&ctrl->s_full[sb]));
          umma_commit_pair(smem_u32(&ctrl->kv_empty[kslot]));
          ++s_j;
          if (s_j == s_nt) umma_commit_pair(smem_u32(&ctrl->q_empty[qb]));   // Q buffer may be refilled
          ++gs;
        }
        if (gs == gp) break;   // end of work and nothing pending
        // ---- 2. PV for the oldest S tile
        {
          if (p_j == 0) {
            const int fi = f_head & 3;
            p_nkeys = ctrl->mma_fifo[fi][0];
            p_slot = ctrl->mma_fifo[fi][1];
            p_kv = static_cast<uint32_t>(ctrl->mma_fifo[fi][2]);
            p_nt = ctrl->mma_fifo[fi][3];
          }
          const int n_keys = p_nkeys;
          const int nt = p_nt;                                  // history tiles, then self tiles
          const uint32_t ob = p_keyed & 1;
          if (p_j == 0 && p_keyed >= 2)   // the epilogue must have drained this O buffer (item p_keyed - 2)
            mbar_wait_cluster(smem_u32(&ctrl->o_empty[ob]), ((p_keyed >> 1) - 1) & 1);
          const uint32_t sb = gp & 1;
          const uint32_t vpos = p_kv + 2 * p_j + 1;
          const uint32_t vslot = vpos % kKvSlots;
          // k-steps of 16 keys: the history's last tile may be short; a self tile has all 128 (P is 0 off the diagonal)
          const int keys_left = n_keys - p_j * kKeys;
          const int ksteps = keys_left > 0 ? (min(kKeys, keys_left) + 15) >> 4 : kKeys / 16;
          const uint32_t v_lo = kv_lo + kLoMN + ((vslot * kHalfBytes) >> 4);
          const uint32_t tp = tmem_base + sb * kKeys;          // P(g, h): packed bf16 pairs at columns 64 h + [0, 32)
          const uint32_t to = tmem_base + 256 + ob * kD;
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            mbar_wait_cluster(smem_u32(&ctrl->p_full[sb][h]), (gp >> 1) & 1);
            if (h == 0) mbar_wait_cluster(smem_u32(&ctrl->kv_full[vslot]), (vpos / kKvSlots) & 1);
            tc_fence_after();
#pragma unroll
            for (int k = 4 * h; k < 4 * h + 4; ++k)
              if (k < ksteps)
                umma_ts_pair(to, tp + h * 64 + (k & 3) * 8, mk_desc(v_lo + k * (2048 >> 4)), kIdescO,
                             (p_j > 0 || k > 0) ? 1u : 0u);
            umma_commit_pair(smem_u32(&ctrl->pv_done[(2 * gp + h) & 3]));
          }
          umma_commit_pair(smem_u32(&ctrl->kv_empty[vslot]));
          ++gp;
          ++p_j;
          if (p_j == nt) {
            umma_commit_pair(smem_u32(&ctrl->o_full[ob]));
            mbar_arrive(smem_u32(&ctrl->item_empty[p_slot]));
            ++f_head;
            ++p_keyed;
            p_j = 0;
          }
        }
      }
    }
    }
    __syncwarp();
  } else if (warp == kHelpWarp0 || warp == kHelpWarp0 + 1) {
    // ================================================================= spare warps
    // (they only hand their registers to the softmax groups)
    setmaxnreg_dec<kOtherRegs>();
  } else if (warp < 8) {
    // ================================================================= softmax groups
    // Both groups work on EVERY key tile of the CTA's 128 rows, two threads per row: group wg owns
    // the tile's columns [64 wg, 64 wg + 64) -- 64 exponentials per thread and tile.  The row's
    // reference maximum is the one quantity the two threads of a row share; it is handed from half
    // tile to half tile (see advance_max below).  Each thread keeps the row sum of its own columns
    // and the reference it is relative to (the epilogue combines the two).  P(g, wg) is written over
    // the group's OWN S columns (packed bf16 at columns 64 wg + [0, 32)), so neither group touches
    // TMEM the other still reads.
    // The two groups' exponential phases run CONCURRENTLY: the two warps that share an SM
    // sub-partition are the two groups' warps of the same 32 rows, one warp alone reaches only half
    // of the MUFU rate (measured: 64 ex2 in ~950 cycles against 512), two together saturate it.
    setmaxnreg_inc<kSoftmaxRegs>();
    const int wg = warp >> 2;
    const int lq = warp & 3;
    const int row = threadIdx.x & 127;       // row of the CTA's tile == TMEM lane
    bool first_step = true;                  // group 0: nobody has published before the kernel's first step
    const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t p_full_addr = mapa_shared(smem_u32(&ctrl->p_full[0][wg]), 0);   // the leader's barriers
    uint32_t g0 = 0;          // global key tiles before the current item
    uint32_t n_keyed = 0;     // keyed items before the current one (O buffer)
    for (uint32_t n = 0;; ++n) {
      const int islot = n & (kItemSlots - 1);
      mbar_wait<7>(smem_u32(&ctrl->item_full[islot]), (n / kItemSlots) & 1);
      const Item it = ctrl->items[islot];
      if (!it.valid) break;
      const int nt_hist = (it.n_keys + kKeys - 1) / kKeys;
      const int nt = nt_hist + (kSelf ? it.n_self : 0);   // history tiles, then one self tile per Q tile with candidates
      const int nh = cands_here(it);
      const int g = row / cpt, cl = row - g * cpt;
      const bool row_valid = cl < nh;
      const uint32_t ob = n_keyed & 1;
      const uint32_t tm_o = tmem_base + lane_base + 256 + ob * kD;   // the row's O accumulator
      // running state, log2 units
      float m_used = -INFINITY;
      float l = 0.f;
      if (nh > 0) {
        // keys this thread's row may see (causal mode; otherwise all of the item's)
        const int lim_row = min(it.n_keys, it.lim0 + static_cast<int>(rank) * cpt + cl);
        const int lim_cta = it.lim0 + static_cast<int>(rank) * cpt;      // ... and the CTA tile's first row
        // Reference maximum of a row.  The 64-key half tiles of an item form ONE sequence of online-softmax steps
        // (tile 0 half 0, tile 0 half 1, tile 1 half 0, ...); group wg owns the steps of half wg.  A step reads the
        // reference its predecessor published, applies the lazy rule (the reference moves only when the step's own
        // maximum exceeds it by more than kTau -- and then this thread alone rescales the whole O row, after every
        // earlier step's PV has completed) and publishes the result for its successor BEFORE its exponentials.
        // Nothing is exchanged symmetrically: group 0 never waits (its predecessor published a whole exponential
        // phase ago), group 1 trails it by the hand-over latency, and the 256-thread barrier with its two shared-
        // memory round trips per tile is gone (measured against it: -2 % on config 3, -4 % on config 5).
        // (Publishing halfway through the exponentials, to put the groups in anti-phase, was slower: a warp alone
        // issues an ex2 every 14 - 16 cycles, two warps of a sub-partition together one every 9.)
        auto advance_max = [&](const float mx_mine, const int j, const uint32_t gidx) {
          float m_prev;
          if (wg == 0) {
            if (!first_step) named_bar_sync(kBarBA + lq, 64);   // (group 1's publication of its previous step)
            first_step = false;
            m_prev = (j == 0) ? -INFINITY : ctrl->ref_sh[1][row];
          } else {
            named_bar_sync(kBarAB + lq, 64);                     // (group 0's publication of this tile's step)
            m_prev = ctrl->ref_sh[0][row];
          }
          if (m_prev != m_used) {          // the other group moved the reference: bring the own row sum along
            l *= ex2_approx(m_used - m_prev);
            m_used = m_prev;
          }
          const float mx = mx_mine * args.scale_log2;
          const float m_new = fmaxf(m_used, mx);
          const bool need = m_new > m_used + kTau;
          if (j == 0 && wg == 0) {
            // nothing accumulated in O yet (the first PV overwrites)
            if (need) m_used = m_new;      // l == 0
          } else if (__any_sync(0xffffffffu, need)) {
            // every earlier step's PV (half-steps < 2 gidx + wg) must have landed in O.  Steps <= 2 gidx - 4 are
            // complete (they were issued before S(gidx), which has been read); a ring of four barriers keeps the
            // parity wait on the step before this one unambiguous even though this path is taken rarely.
            const uint32_t hp = 2 * gidx + wg - 1;
            mbar_wait<10>(smem_u32(&ctrl->pv_done[hp & 3]), (hp >> 2) & 1);
            tc_fence_after();
            const float alpha = need ? ex2_approx(m_used - m_new) : 1.0f;
#pragma unroll 1
            for (int c0 = 0; c0 < kD; c0 += 16) {
              uint32_t orr[16];
              tmem_ld16(tm_o + c0, orr);
              tmem_wait_ld_regs(orr);
#pragma unroll
              for (int c = 0; c < 16; ++c) orr[c] = __float_as_uint(__uint_as_float(orr[c]) * alpha);
              tmem_st16(tm_o + c0, orr);
            }
            tmem_wait_st();
            l *= alpha;
            if (need) m_used = m_new;
          }
        };
        auto publish = [&]() {
          ctrl->ref_sh[wg][row] = m_used;
          named_bar_arrive((wg == 0 ? kBarAB : kBarBA) + lq, 64);
        };
        // One 128-key tile.  Tiles that need masking (the item's last tile: history tail; causal mode: the
        // tiles that reach past the diagonal) are a separate instantiation so that the steady-state loop
        // body stays small.
        auto step = [&](const int j, auto last_tag) {
          constexpr bool kLast = decltype(last_tag)::value;
          const uint32_t gidx = g0 + j;
          const uint32_t sb = gidx & 1;
          const uint32_t tm_s = tmem_base + lane_base + sb * kKeys + wg * 64;   // own columns of S(g)
          mbar_wait<9>(smem_u32(&ctrl->s_full[sb]), (gidx >> 1) & 1);
          tc_fence_after();
          uint32_t sr[64];
          tmem_ld32(tm_s, &sr[0]);
          tmem_ld32(tm_s + 32, &sr[32]);
          tmem_wait_ld_regs(sr);
          const int keys_mine = kLast ? lim_row - j * kKeys - wg * 64 : 64;   // valid keys among this thread's columns
          if (kLast) {
#pragma unroll
            for (int c = 0; c < 64; ++c)
              if (c >= keys_mine) sr[c] = 0xff800000u;  // -inf
          }
          float mxa = fmax3(__uint_as_float(sr[0]), __uint_as_float(sr[1]), __uint_as_float(sr[2]));
          float mxb = fmax3(__uint_as_float(sr[3]), __uint_as_float(sr[4]), __uint_as_float(sr[5]));
          float mxc = fmaxf(__uint_as_float(sr[6]), __uint_as_float(sr[7]));
          float mxd = -INFINITY;
#pragma unroll
          for (int c = 8; c < 64; c += 8) {
            mxa = fmax3(mxa, __uint_as_float(sr[c + 0]), __uint_as_float(sr[c + 1]));
            mxb = fmax3(mxb, __uint_as_float(sr[c + 2]), __uint_as_float(sr[c + 3]));
            mxc = fmax3(mxc, __uint_as_float(sr[c + 4]), __uint_as_float(sr[c + 5]));
            mxd = fmax3(mxd, __uint_as_float(sr[c + 6]), __uint_as_float(sr[c + 7]));
          }
          const float mx_mine = fmaxf(fmaxf(mxa, mxb), fmaxf(mxc, mxd));
          advance_max(mx_mine, j, gidx);
          publish();
          float2 sumA = make_float2(0.f, 0.f), sumB = make_float2(0.f, 0.f);
          // (a row that has seen no key yet -- causal mode with more candidates than keys -- keeps m = -inf:
          // subtract 0 instead, its logits are all -inf and its weights 0)
          const float m_sub = (kLast && m_used == -INFINITY) ? 0.f : m_used;
          const float2 c2 = make_float2(args.scale_log2, args.scale_log2);
          float2 nm2 = make_float2(-m_sub, -m_sub);
#pragma unroll
          for (int c0 = 0; c0 < 64; c0 += 32) {
            uint32_t pr[16];
            // masked tile: 32 columns that no row of the warp can see cost no exponentials (the history's last
            // tile is on average half empty: ~40 % of its MUFU work)
            if (kLast && __all_sync(0xffffffffu, keys_mine <= c0)) {
#pragma unroll
              for (int c = 0; c < 16; ++c) pr[c] = 0u;
              tmem_st16(tm_s + (c0 >> 1), pr);
              continue;
            }
#pragma unroll
            for (int c = 0; c < 32; c += 4) {
              const float2 x01 = ffma2(make_float2(__uint_as_float(sr[c0 + c + 0]),
                                                   __uint_as_float(sr[c0 + c + 1])), c2, nm2);
              const float2 x23 = ffma2(make_float2(__uint_as_float(sr[c0 + c + 2]),
                                                   __uint_as_float(sr[c0 + c + 3])), c2, nm2);
              const float p0 = ex2_approx(x01.x), p1 = ex2_approx(x01.y);
              const float p2 = ex2_approx(x23.x), p3 = ex2_approx(x23.y);
              const uint32_t w01 = pack_bf16x2(p0, p1), w23 = pack_bf16x2(p2, p3);
              pr[(c >> 1) + 0] = w01;
              pr[(c >> 1) + 1] = w23;
              // the row sum adds the bf16-ROUNDED weights: out stays a convex combination of V rows
              add_bf16x2_f32(sumA.x, sumA.y, w01);
              add_bf16x2_f32(sumB.x, sumB.y, w23);
            }
            // P(g, wg): packed bf16 pairs over the group's own S columns
            tmem_st16(tm_s + (c0 >> 1), pr);
          }
          l += (sumA.x + sumA.y) + (sumB.x + sumB.y);
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(p_full_addr + sb * 16);
        };
        // Self tile t = j - nt_hist: its keys are Q tile t's own rows under the identity block of the mask
        // (PAPER.md:198): row r of CTA t sees key r, every other (row, key) pair of the tile is masked.  One logit,
        // one exponential and one non-zero P entry per row: the row's thread whose columns hold the diagonal
        // (group row / 64) picks S[r][r] out of the 32 columns its warp's diagonal lies in; everything else in P is 0.
        auto self_step = [&](const int j) {
          const uint32_t gidx = g0 + j;
          const uint32_t sb = gidx & 1;
          const uint32_t tm_s = tmem_base + lane_base + sb * kKeys + wg * 64;
          mbar_wait<9>(smem_u32(&ctrl->s_full[sb]), (gidx >> 1) & 1);
          tc_fence_after();
          const bool tile_mine = (j - nt_hist) == static_cast<int>(rank);
          const bool diag_warp = tile_mine && ((warp >> 1) & 1) == wg;       // warp-uniform: rows [32 (warp & 3), +32)
          const uint32_t dcol = (warp & 1) * 32;                              // ... have their diagonal at these columns
          float x = -INFINITY;
          if (diag_warp) {
            uint32_t sr[32];
            tmem_ld32(tm_s + dcol, sr);
            tmem_wait_ld_regs(sr);
            uint32_t v = 0;
#pragma unroll
            for (int c = 0; c < 32; ++c) v = (c == lane) ? sr[c] : v;
            if (row_valid) x = __uint_as_float(v);
          }
          advance_max(x, j, gidx);
          publish();
          const float m_sub = (m_used == -INFINITY) ? 0.f : m_used;
          const float w = ex2_approx(fmaf(x, args.scale_log2, -m_sub));      // 0 for every thread without a diagonal
          const uint32_t wb = pack_bf16x2(w, 0.f);                            // bf16(w) in the low half
          l += __uint_as_float(wb << 16);
          const uint32_t val = (lane & 1) ? (wb << 16) : wb;                  // key row & 63 = dcol + lane: packed column (dcol + lane) / 2
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            uint32_t z[16];
            const bool here = diag_warp && hh == (warp & 1);
#pragma unroll
            for (int i = 0; i < 16; ++i) z[i] = (here && i == (lane >> 1)) ? val : 0u;
            tmem_st16(tm_s + hh * 16, z);
          }
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(p_full_addr + sb * 16);
        };
        for (int j = 0; j < nt_hist; ++j) {
          if (j == nt_hist - 1 || (j + 1) * kKeys > lim_cta) step(j, cuda::std::true_type{});
          else step(j, cuda::std::false_type{});
        }
        if constexpr (kSelf) {
          for (int j = nt_hist; j < nt; ++j) self_step(j);
        }
        // hand the row's final state to the epilogue: each group's partial sum and the reference it is relative
        // to (group 1's is the last step's, i.e. the one O is in; the epilogue brings group 0's sum to it)
        ctrl->epi_l[islot][wg][row] = l;
        ctrl->epi_m[islot][wg][row] = m_used;
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->l_ready[islot]));
      } else {
        // this CTA's tile has no valid row for this item: keep the pair's barriers moving
        for (int j = 0; j < nt; ++j) {
          const uint32_t gidx = g0 + j;
          const uint32_t sb = gidx & 1;
          mbar_wait<9>(smem_u32(&ctrl->s_full[sb]), (gidx >> 1) & 1);
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(p_full_addr + sb * 16);
        }
      }
      if (nt > 0) {
        g0 += nt;
        ++n_keyed;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->item_empty[islot]));
    }
  } else {
    // ================================================================= epilogue group (a7)
    setmaxnreg_dec<kEpilogueRegs>();
    const int ew = warp - kEpiWarp0;                     // TMEM lane quarter of this warp
    const uint32_t lane_base = static_cast<uint32_t>(ew * 32) << 16;
    const uint32_t stage = epi_smem + ew * kEpiWarpBytes;
    const uint32_t o_empty_addr = mapa_shared(smem_u32(&ctrl->o_empty[0]), 0);   // the leader's barriers
    uint32_t n_keyed = 0;
    uint32_t lr_par = 0;      // bit s: parity of the next l_ready[s] phase to wait for
    for (uint32_t n = 0;; ++n) {
      const int islot = n & (kItemSlots - 1);
      mbar_wait<11>(smem_u32(&ctrl->item_full[islot]), (n / kItemSlots) & 1);
      const Item it = ctrl->items[islot];
      if (!it.valid) break;
      const int nt = (it.n_keys + kKeys - 1) / kKeys + it.n_self;
      const int nh = cands_here(it);
      const uint32_t ob = n_keyed & 1;
      if (nh > 0) {
        mbar_wait<12>(smem_u32(&ctrl->l_ready[islot]), (lr_par >> islot) & 1);
        lr_par ^= 1u << islot;
      }
      if (nt > 0) {
        mbar_wait<13>(smem_u32(&ctrl->o_full[ob]), (n_keyed >> 1) & 1);
        tc_fence_after();
      }
      if (nh > 0) {
        const int row = ew * 32 + lane;                  // row of this thread within the tile
        const float m0 = ctrl->epi_m[islot][0][row], m1 = ctrl->epi_m[islot][1][row];
        const float l0 = ctrl->epi_l[islot][0][row], l1 = ctrl->epi_l[islot][1][row];
        const float lsum = (m0 == m1) ? l0 + l1 : fmaf(l0, ex2_approx(m0 - m1), l1);
        const float inv = partial ? 1.0f : (lsum > 0.f ? 1.0f / lsum : 0.f);
        if (partial) {     // split-K: the row's state (reference maximum, row sum) beside the unnormalised O
          const int g_r = row / cpt, cl_r = row - g_r * cpt;
          if (cl_r < nh) {
            const size_t prow = ((static_cast<size_t>(it.layer) * args.total_q + it.c0 + rank * cpt + cl_r) * args.H_q +
                                 it.hkv * G + g_r) * args.num_splits + it.split;
            args.part_ml[prow * 2 + 0] = m1;
            args.part_ml[prow * 2 + 1] = lsum;
          }
        }
        const float2 sc2 = make_float2(inv, inv);
        const int cand0 = it.c0 + static_cast<int>(rank) * cpt;       // first candidate of this CTA's tile
        const size_t lrow0 = static_cast<size_t>(it.layer) * args.total_q;
        const uint32_t tm_o = tmem_base + lane_base + 256 + ob * kD;
        // the warp's 32 rows are 32 consecutive candidates of one query head when cpt >= 32
        const int g_w = (ew * 32) / cpt, cl_w = (ew * 32) - g_w * cpt;
        const bool warp_full = cpt >= 32 && cl_w + 32 <= nh;
        if (args.out_tma && !partial && nt > 0 && warp_full) {
          // all 32 rows valid: each 32 x 32 block leaves through one TMA store from a swizzled box
          const int grow = static_cast<int>(lrow0) + cand0 + cl_w;
          const int gcol = (it.hkv * G + g_w) * kD;
          const uint32_t sw_row = stage + lane * 128;
          uint32_t orr[32];
          tmem_ld32(tm_o, orr);
#pragma unroll 1
          for (int c0 = 0; c0 < kD; c0 += 32) {
            tmem_wait_ld_regs(orr);
            if (c0 + 32 == kD) {
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(o_empty_addr + ob * 8);
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
            if (c0 + 32 < kD) tmem_ld32(tm_o + c0 + 32, orr);   // next block: overlaps the store hand-off
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&tmap_out, stage, gcol + c0, grow);
              bulk_commit();
            }
          }
        } else {
          // general path: ragged rows, split-K partials, key-less items, G > 4
          if (lane == 0) bulk_wait_read_all();   // a TMA store of an earlier item may still read the block
          __syncwarp();
          // transposed read-back: 8 lanes cover one row's 128-byte line, 4 rows per access
          const int rr = lane >> 3, cq = lane & 7;
          const uint32_t st_w = stage + lane * kEpiRowBytes;
          const uint32_t st_r = stage + rr * kEpiRowBytes + cq * 16;
#pragma unroll 1
          for (int c0 = 0; c0 < kD; c0 += 32) {
            uint32_t orr[32];
            if (nt > 0) {
              tmem_ld32(tm_o + c0, orr);
              tmem_wait_ld_regs(orr);
              if (c0 + 32 == kD) {
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(o_empty_addr + ob * 8);
              }
            } else {
#pragma unroll
              for (int c = 0; c < 32; ++c) orr[c] = 0u;
            }
#pragma unroll
            for (int c = 0; c < 32; c += 8) {
              float o[8];
#pragma unroll
              for (int k = 0; k < 8; ++k) o[k] = __uint_as_float(orr[c + k]) * inv;
              sts128(st_w + c * 4, __float_as_uint(o[0]), __float_as_uint(o[1]), __float_as_uint(o[2]),
                     __float_as_uint(o[3]));
              sts128(st_w + c * 4 + 16, __float_as_uint(o[4]), __float_as_uint(o[5]), __float_as_uint(o[6]),
                     __float_as_uint(o[7]));
            }
            __syncwarp();
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const int r2 = ew * 32 + 4 * k + rr;       // tile row this lane group stores
              const int g2 = r2 / cpt, cl2 = r2 - g2 * cpt;
              if (cl2 < nh) {
                const size_t orow = (lrow0 + cand0 + cl2) * args.H_q + it.hkv * G + g2;
                float* dst = partial ? args.part_o + (orow * args.num_splits + it.split) * kD
                                     : args.out + orow * kD;
                stg128_stream(dst + c0 + cq * 4, lds128(st_r + k * (4 * kEpiRowBytes)));
              }
            }
            __syncwarp();
          }
        }
      } else if (nt > 0) {
        // no valid row in this CTA's tile: the accumulator is handed straight back
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(o_empty_addr + ob * 8);
      }
      if (nt > 0) ++n_keyed;
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
  cluster_sync_all();      // the peer may still signal this CTA's barriers / read its shared memory
  if (warp == kMmaWarp) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base, 512);
  }
}

}  // namespace pair
}  // namespace upr
