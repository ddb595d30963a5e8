// sched_kernel.cuh -- step a0 on the device: the work-list tables of one forward call.
//
// One small CTA per call (graph-capturable, no host read of any device table):
//   order[i]    users sorted by history length, LONGEST FIRST (long, ragged
//               histories are what bounds the ranking pass), ties by user index;
//   iprefix[i]  exclusive prefix sum, in that order, of the work items one layer of user order[i]
//               contributes: ceil(C_b / cands_per_block) * H_kv * num_splits;  iprefix[B] = W;
//   rowoff[b]   exclusive prefix sum over USER INDEX of round_up(L_b, 16): the row offsets of the
//               packed cache (the same integers upr_kv_cache_layout returns on the host);
//   counter     the dynamic scheduler's work counter, reset to 0.
// Work item idx (handed out by the counter) is then: i = the position with
// n_layers * iprefix[i] <= idx < n_layers * iprefix[i+1]; the layers of one user are adjacent, so
// the order is longest-first over (user, layer) pairs across the whole call.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace upr {

constexpr int kSchedThreads = 1024;
constexpr int kSchedSortMax = 4096;   // larger batches keep the user order (no sort)

struct SchedArgs {
  const int32_t* seq_lens;
  const int32_t* cand_offsets;
  unsigned int* counter;
  int32_t* iprefix;   // [B + 1]
  int32_t* order;     // [B]
  int32_t* rowoff;    // [B + 1]
  int B, H_kv, num_splits, cands_per_block;
};

__global__ void __launch_bounds__(kSchedThreads, 1) upr_schedule_kernel(const SchedArgs a) {
  __shared__ uint32_t keys[kSchedSortMax];
  __shared__ int wsum_w[32], wsum_r[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) *a.counter = 0u;

  // ---- 1. order: bitonic sort of (max_len - L_b, b) keys, ascending = longest first
  if (a.B <= kSchedSortMax) {
    int n = 1;
    while (n < a.B) n <<= 1;
    for (int i = tid; i < n; i += kSchedThreads) {
      uint32_t key = 0xFFFFFFFFu;
      if (i < a.B) {
        const int L = min(max(__ldg(a.seq_lens + i), 0), 0xFFFFF);
        key = (static_cast<uint32_t>(0xFFFFF - L) << 12) | static_cast<uint32_t>(i);
      }
      keys[i] = key;
    }
    __syncthreads();
    for (int k = 2; k <= n; k <<= 1) {
      for (int j = k >> 1; j > 0; j >>= 1) {
        for (int i = tid; i < n; i += kSchedThreads) {
          const int ixj = i ^ j;
          if (ixj > i) {
            const uint32_t x = keys[i], y = keys[ixj];
            const bool up = (i & k) == 0;
            if ((x > y) == up) {
              keys[i] = y;
              keys[ixj] = x;
            }
          }
        }
        __syncthreads();
      }
    }
    for (int i = tid; i < a.B; i += kSchedThreads) a.order[i] = static_cast<int32_t>(keys[i] & 0xFFFu);
  } else {
    for (int i = tid; i < a.B; i += kSchedThreads) a.order[i] = i;
  }
  __syncthreads();   // order[] (global) written by this block is visible to it

  // ---- 2. the two prefix sums: a contiguous chunk per thread, block scan of the chunk sums
  const int per = (a.B + kSchedThreads - 1) / kSchedThreads;
  const int lo = min(a.B, tid * per), hi = min(a.B, lo + per);
  auto items_of = [&](int b) {
    const int C = __ldg(a.cand_offsets + b + 1) - __ldg(a.cand_offsets + b);
    return (C + a.cands_per_block - 1) / a.cands_per_block * a.H_kv * a.num_splits;
  };
  auto rows_of = [&](int b) { return (max(__ldg(a.seq_lens + b), 0) + 15) / 16 * 16; };
  int sw = 0, sr = 0;
  for (int i = lo; i < hi; ++i) {
    sw += items_of(a.order[i]);
    sr += rows_of(i);
  }
  int iw = sw, ir = sr;   // inclusive scans over threads
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int tw = __shfl_up_sync(0xffffffffu, iw, o), tr = __shfl_up_sync(0xffffffffu, ir, o);
    if (lane >= o) {
      iw += tw;
      ir += tr;
    }
  }
  if (lane == 31) {
    wsum_w[warp] = iw;
    wsum_r[warp] = ir;
  }
  __syncthreads();
  if (warp == 0) {
    int vw = wsum_w[lane], vr = wsum_r[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int tw = __shfl_up_sync(0xffffffffu, vw, o), tr = __shfl_up_sync(0xffffffffu, vr, o);
      if (lane >= o) {
        vw += tw;
        vr += tr;
      }
    }
    wsum_w[lane] = vw;
    wsum_r[lane] = vr;
  }
  __syncthreads();
  int base_w = iw - sw + (warp > 0 ? wsum_w[warp - 1] : 0);
  int base_r = ir - sr + (warp > 0 ? wsum_r[warp - 1] : 0);
  for (int i = lo; i < hi; ++i) {
    a.iprefix[i] = base_w;
    a.rowoff[i] = base_r;
    base_w += items_of(a.order[i]);
    base_r += rows_of(i);
  }
  if (tid == kSchedThreads - 1) {
    a.iprefix[a.B] = wsum_w[31];
    a.rowoff[a.B] = wsum_r[31];
  }
}

}  // namespace upr
