// upr_api.cu -- C ABI of libupr (include/upr.h): argument checks, tensor-map encoding, launches.
// No torch types, no host synchronisation, no device allocation.
#include <cuda.h>
#include <mutex>
#include <vector>
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <atomic>

#include "../../include/upr.h"
#include "attn2_kernel.cuh"
#include "attn_kernel.cuh"
#include "linear2_kernel.cuh"
#include "linear_kernel.cuh"
#include "pack_kernels.cuh"
#include "sched_kernel.cuh"
#include "tail_kernels.cuh"

namespace {

thread_local char g_err[512] = "";
thread_local int g_launches = 0;
thread_local const char* g_kernel = "";

upr_status fail(upr_status s, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return s;
}

#define UPR_CUDA_CHECK(expr)                                                              \
  do {                                                                                    \
    cudaError_t e_ = (expr);                                                              \
    if (e_ != cudaSuccess)                                                                \
      return fail(UPR_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e_));          \
  } while (0)

int elem_bytes(int dtype) { return dtype == UPR_F32 ? 4 : dtype == UPR_BF16 ? 2 : 1; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  // the driver entry point is process-wide and immutable; a racing first call stores the same value
  static std::atomic<EncodeTiledFn> fn{nullptr};
  EncodeTiledFn f = fn.load(std::memory_order_acquire);
  if (f == nullptr) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) ==
            cudaSuccess &&
        qres == cudaDriverEntryPointSuccess) {
      f = reinterpret_cast<EncodeTiledFn>(p);
      fn.store(f, std::memory_order_release);
    }
  }
  return f;
}

// 2-D bf16 view [rows, d] of a packed cache or of the pool; box = [box_rows x 64 cols], 128-byte
// swizzle.  rows = 0: the extent is left unbounded (a packed cache's R depends on device-resident
// seq_lens the host never reads; the layout contract guarantees UPR_TAIL_ROWS of slack); rows > 0
// (pool, or a caller-stated buffer size): boxes are clipped there, rows beyond it read as zeros.
upr_status make_kv_tmap(CUtensorMap* m, const void* base, int d, long long rows, int box_rows = 128) {
  EncodeTiledFn enc = get_encode_fn();
  if (enc == nullptr) return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t gdim[2] = {static_cast<cuuint64_t>(d),
                        rows > 0 ? static_cast<cuuint64_t>(rows) : static_cast<cuuint64_t>(1) << 31};
  cuuint64_t gstride[1] = {static_cast<cuuint64_t>(d) * 2};
  cuuint32_t box[2] = {64, static_cast<cuuint32_t>(box_rows)};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstride,
                   box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return UPR_OK;
}

// Per-device facts, queried on every call (two cheap runtime calls): nothing is cached across
// devices or threads, so a process may use the library on any number of devices and threads.
int sm_count() {
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return 0;
  return n;
}

upr_status check_device() {
  int dev = 0, major = 0;
  UPR_CUDA_CHECK(cudaGetDevice(&dev));
  UPR_CUDA_CHECK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  if (major != 10) return fail(UPR_ERR_UNSUPPORTED, "libupr requires an sm_100a (B200) device");
  return UPR_OK;
}

constexpr size_t kCounterBytes = 256;

int kv_heads(const upr_attn_params* p) { return p->H_kv > 0 ? p->H_kv : p->H; }

// Which attention kernel runs these arguments.  The CTA-pair kernel (attn2_kernel.cuh) takes the
// tensor-bound shapes: bf16 q and K/V, d = 128, a workspace (the extended entry point), query
// groups of 1/2/4/8, and on average more than one 128-row tile of (candidate, head) rows per user
// -- below that its second CTA would idle and the 1-CTA kernel streams K/V at the HBM rate.
bool pair_capable(const upr_attn_params* p) {
  const int hkv = kv_heads(p);
  const int G = hkv > 0 ? p->H / hkv : 0;
  return p->d == 128 && p->kv_dtype == UPR_BF16 && p->q_dtype == UPR_BF16 &&
         (G == 1 || G == 2 || G == 4 || G == 8) &&
         static_cast<long long>(p->n_layers) * p->total_q < (1LL << 31);
}

constexpr bool kPairInAuto = true;

bool use_pair(const upr_attn_params* p, bool have_workspace) {
  if (!have_workspace || p->kernel == UPR_KERNEL_SINGLE || !pair_capable(p)) return false;
  if (p->kernel == UPR_KERNEL_PAIR || p->causal) return true;
  if (!kPairInAuto) return false;
  const int G = p->H / kv_heads(p);
  if (G > 1) return true;   // grouped queries exist only in the pair kernel
  return p->B > 0 && static_cast<long long>(p->total_q) * G > 128LL * p->B;
}

int pick_splits(const upr_attn_params* p, bool pair) {
  if (p->causal) return 1;
  if (p->num_splits >= 1) return p->num_splits;
  // heuristic: split the history when the (user, head, q-block) items cannot fill the SMs
  if (p->max_seq_len <= 0 || p->total_q <= 0 || p->B <= 0) return 1;
  const int sms = sm_count() > 0 ? sm_count() : 148;
  const int units = pair ? sms / 2 : sms;   // CTA pairs or CTAs
  const int G = p->H / kv_heads(p);
  const int rows_per_block = upr::kQBlock / (pair ? G : 1);   // candidates per 256-row block
  const long long blocks = (p->total_q + rows_per_block - 1) / rows_per_block + p->B / 2;
  const long long items = blocks * kv_heads(p) * p->n_layers;
  const int tiles = (p->max_seq_len + upr::kTileN - 1) / upr::kTileN;
  if (items >= 2LL * units || tiles < 4) return 1;
  long long want = (2LL * units + items - 1) / items;
  long long cap = tiles / 2;  // at least two tiles per split
  long long ns = want < cap ? want : cap;
  if (ns > 16) ns = 16;
  return ns < 1 ? 1 : static_cast<int>(ns);
}

// workspace: [scheduler counter block][work-list tables: iprefix[B+1], order[B], rowoff[B+1]][split-K partials]
size_t tables_bytes(int B) { return (static_cast<size_t>(3) * (B + 1) * sizeof(int32_t) + 255) / 256 * 256; }

upr_status validate(const upr_attn_params* p) {
  if (p == nullptr) return fail(UPR_ERR_INVALID_ARG, "params is NULL");
  if (p->B < 0 || p->H <= 0 || p->n_layers <= 0 || p->total_q < 0)
    return fail(UPR_ERR_INVALID_ARG, "negative or zero size (B=%d H=%d n_layers=%d total_q=%lld)",
                p->B, p->H, p->n_layers, (long long)p->total_q);
  if (p->d != 64 && p->d != 128)
    return fail(UPR_ERR_UNSUPPORTED, "head dim d=%d unsupported (64 or 128)", p->d);
  if (p->kv_dtype != UPR_BF16 && p->kv_dtype != UPR_FP8_E4M3 && p->kv_dtype != UPR_F32 &&
      p->kv_dtype != UPR_FP8_E4M3_USER)
    return fail(UPR_ERR_UNSUPPORTED, "kv_dtype %d unsupported (f32, bf16 or fp8 e4m3)", p->kv_dtype);
  if (p->q_dtype != UPR_BF16 && p->q_dtype != UPR_F32)
    return fail(UPR_ERR_UNSUPPORTED, "q_dtype %d unsupported (bf16 or f32)", p->q_dtype);
  if (p->B > 0 && p->total_q > 0 &&
      (!p->q || !p->k_cache || !p->v_cache || !p->seq_lens || !p->cand_offsets || !p->out))
    return fail(UPR_ERR_INVALID_ARG, "NULL tensor pointer");
  if ((p->k_self == nullptr) != (p->v_self == nullptr))
    return fail(UPR_ERR_INVALID_ARG, "k_self and v_self must both be set or both be NULL");
  if (p->sm_scale < 0.f || isnan(p->sm_scale))
    return fail(UPR_ERR_INVALID_ARG, "sm_scale must be >= 0 (0 selects 1/sqrt(d))");
  if (p->num_splits < 0 || p->num_splits > 64)
    return fail(UPR_ERR_INVALID_ARG, "num_splits=%d out of range [0,64]", p->num_splits);
  if (p->H_kv < 0 || (p->H_kv > 0 && p->H % p->H_kv != 0))
    return fail(UPR_ERR_INVALID_ARG, "H_kv=%d must divide H=%d", p->H_kv, p->H);
  const int hkv = p->H_kv > 0 ? p->H_kv : p->H;
  if (p->kv_bytes < 0 || p->kv_rows < 0) return fail(UPR_ERR_INVALID_ARG, "negative kv_bytes / kv_rows");
  const long long row_bytes = static_cast<long long>(p->d) * elem_bytes(p->kv_dtype);
  if (p->kv_source == UPR_KV_POOL) {
    if (p->kv_dtype != UPR_BF16)
      return fail(UPR_ERR_UNSUPPORTED, "the pool is bf16 (PAPER.md:202): kv_source = UPR_KV_POOL needs kv_dtype = UPR_BF16");
    if (p->pool_slots <= 0 || p->pool_n_max <= 0)
      return fail(UPR_ERR_INVALID_ARG, "bad pool shape S=%d n=%d", p->pool_slots, p->pool_n_max);
    if (p->B > 0 && p->slot_ids == nullptr) return fail(UPR_ERR_INVALID_ARG, "slot_ids is NULL");
    const long long rows = static_cast<long long>(p->n_layers) * p->pool_slots * hkv * p->pool_n_max;
    if (rows >= (1LL << 31))
      return fail(UPR_ERR_UNSUPPORTED, "pool has too many rows for 32-bit TMA coordinates");
    if (p->kv_bytes > 0 && p->kv_bytes < rows * row_bytes)
      return fail(UPR_ERR_INVALID_ARG, "pool buffer too short: %lld bytes stated, %lld needed",
                  (long long)p->kv_bytes, rows * row_bytes);
  } else if (p->kv_source == UPR_KV_PACKED) {
    if (p->kv_bytes > 0 && p->kv_rows > 0) {
      const long long need =
          (static_cast<long long>(p->n_layers) * hkv * p->kv_rows + UPR_TAIL_ROWS) * row_bytes;
      if (p->kv_bytes < need)
        return fail(UPR_ERR_INVALID_ARG, "cache buffer too short: %lld bytes stated, %lld needed",
                    (long long)p->kv_bytes, need);
    }
  } else {
    return fail(UPR_ERR_INVALID_ARG, "kv_source %d unknown", p->kv_source);
  }
  return UPR_OK;
}

template <int D, int KV>
upr_status launch_attn(const upr::AttnArgs& a, const CUtensorMap& tk, const CUtensorMap& tv,
                       const CUtensorMap& to, const CUtensorMap& tq, int grid, cudaStream_t st) {
  using Cfg = upr::AttnCfg<D, KV>;
  // per call: the attribute is per device (and per context), the call costs about a microsecond
  UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::upr_attn_fwd_kernel<D, KV>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemTotal));
  upr::upr_attn_fwd_kernel<D, KV><<<grid, upr::kAttnThreads, Cfg::kSmemTotal, st>>>(tk, tv, to, tq, a);
  UPR_CUDA_CHECK(cudaGetLastError());
  return UPR_OK;
}

template <int D>
upr_status launch_attn_d(int kv_dtype, const upr::AttnArgs& a, const CUtensorMap& tk,
                         const CUtensorMap& tv, const CUtensorMap& to, const CUtensorMap& tq, int grid,
                         cudaStream_t st) {
  switch (kv_dtype) {
    case UPR_BF16: return launch_attn<D, upr::KV_BF16>(a, tk, tv, to, tq, grid, st);
    case UPR_FP8_E4M3:
    case UPR_FP8_E4M3_USER: return launch_attn<D, upr::KV_FP8>(a, tk, tv, to, tq, grid, st);
    default: return launch_attn<D, upr::KV_F32>(a, tk, tv, to, tq, grid, st);
  }
}

// 2-D tensor map [rows, cols] of a row-major candidate-side tensor (q: bf16, out: fp32)
bool make_cand_tmap(CUtensorMap* m, CUtensorMapDataType dt, int elem, const void* base, long long rows,
                    long long cols, int box_cols, int box_rows, CUtensorMapL2promotion promo) {
  EncodeTiledFn enc = get_encode_fn();
  if (enc == nullptr) return false;
  cuuint64_t gdim[2] = {static_cast<cuuint64_t>(cols), static_cast<cuuint64_t>(rows)};
  cuuint64_t gstride[1] = {static_cast<cuuint64_t>(cols) * elem};
  cuuint32_t box[2] = {static_cast<cuuint32_t>(box_cols), static_cast<cuuint32_t>(box_rows)};
  cuuint32_t estr[2] = {1, 1};
  return enc(m, dt, 2, const_cast<void*>(base), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

upr_status launch_combine(const float* part_o, const float* part_ml, float* out, long long out_rows, int ns,
                          int d, cudaStream_t st) {
  long long blocks = (out_rows + 7) / 8;
  int cgrid = static_cast<int>(blocks < sm_count() * 8LL ? blocks : sm_count() * 8LL);
  if (d == 64)
    upr::upr_combine_kernel<64><<<cgrid, 256, 0, st>>>(part_o, part_ml, out, out_rows, ns);
  else
    upr::upr_combine_kernel<128><<<cgrid, 256, 0, st>>>(part_o, part_ml, out, out_rows, ns);
  UPR_CUDA_CHECK(cudaGetLastError());
  return UPR_OK;
}

// rows of the 2-D [rows, d] view of the K / V storage the tensor maps may touch (0 = unbounded)
long long kv_view_rows(const upr_attn_params* p) {
  long long rows = 0;
  if (p->kv_source == UPR_KV_POOL)
    rows = static_cast<long long>(p->n_layers) * p->pool_slots * kv_heads(p) * p->pool_n_max;
  else if (p->kv_bytes > 0)
    rows = p->kv_bytes / (static_cast<long long>(p->d) * 2);
  return rows >= (1LL << 31) ? 0 : rows;
}

// ---- the CTA-pair kernel (bf16, d = 128): schedule tables -> attention [-> combine]
upr_status run_attn_pair(const upr_attn_params* p, int ns, cudaStream_t st) {
  const int hkv = kv_heads(p), G = p->H / hkv;
  uint8_t* ws = static_cast<uint8_t*>(p->workspace);
  int32_t* tables = reinterpret_cast<int32_t*>(ws + kCounterBytes);
  const long long out_rows = static_cast<long long>(p->n_layers) * p->total_q * p->H;

  upr::SchedArgs sa;
  sa.seq_lens = p->seq_lens;
  sa.cand_offsets = p->cand_offsets;
  sa.counter = reinterpret_cast<unsigned int*>(ws);
  sa.iprefix = tables;
  sa.order = tables + (p->B + 1);
  sa.rowoff = tables + 2 * (p->B + 1);
  sa.B = p->B;
  sa.H_kv = hkv;
  sa.num_splits = ns;
  sa.cands_per_block = 2 * (128 / G);
  upr::upr_schedule_kernel<<<1, upr::kSchedThreads, 0, st>>>(sa);
  UPR_CUDA_CHECK(cudaGetLastError());

  upr::pair::Args a;
  memset(&a, 0, sizeof(a));
  a.q = p->q;
  a.k_self = p->k_self;
  a.v_self = p->v_self;
  a.out = p->out;
  a.seq_lens = p->seq_lens;
  a.cand_offsets = p->cand_offsets;
  a.slot_ids = (p->kv_source == UPR_KV_POOL) ? p->slot_ids : nullptr;
  a.iprefix = sa.iprefix;
  a.order = sa.order;
  a.rowoff = sa.rowoff;
  a.counter = sa.counter;
  a.B = p->B;
  a.H_q = p->H;
  a.H_kv = hkv;
  a.G = G;
  a.cpt = 128 / G;
  a.n_layers = p->n_layers;
  a.num_splits = ns;
  a.pool_S = p->pool_slots;
  a.pool_n = p->pool_n_max;
  a.total_q = static_cast<int>(p->total_q);
  a.causal = p->causal ? 1 : 0;
  const float sm = p->sm_scale > 0.f ? p->sm_scale : 1.0f / sqrtf(static_cast<float>(p->d));
  a.scale_log2 = sm * 1.4426950408889634f;
  if (ns > 1) {
    a.part_o = reinterpret_cast<float*>(ws + kCounterBytes + tables_bytes(p->B));
    a.part_ml = a.part_o + static_cast<size_t>(out_rows) * ns * p->d;
  }

  CUtensorMap tk, tv, tq, to, tks, tvs;
  memset(&to, 0, sizeof(to));
  const long long rows = kv_view_rows(p);
  upr_status s = make_kv_tmap(&tk, p->k_cache, p->d, rows, /*box_rows=*/64);    // K half: 64 keys x 64 d boxes
  if (s != UPR_OK) return s;
  s = make_kv_tmap(&tv, p->v_cache, p->d, rows, /*box_rows=*/128);              // V half: 128 keys x 64 d
  if (s != UPR_OK) return s;
  const long long cand_rows = static_cast<long long>(p->n_layers) * p->total_q;
  const long long cand_cols = static_cast<long long>(p->H) * p->d;
  if (!make_cand_tmap(&tq, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p->q, cand_rows, cand_cols, 64, a.cpt,
                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B))
    return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled failed for q");
  // the candidates' own keys / values enter as one more key tile per Q tile, in the Q tile's row order
  tks = tq;
  tvs = tq;
  if (p->k_self != nullptr) {
    if ((reinterpret_cast<uintptr_t>(p->k_self) & 15) || (reinterpret_cast<uintptr_t>(p->v_self) & 15))
      return fail(UPR_ERR_INVALID_ARG, "k_self / v_self must be 16-byte aligned");
    if (!make_cand_tmap(&tks, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p->k_self, cand_rows, cand_cols, 64,
                        a.cpt < 64 ? a.cpt : 64, CU_TENSOR_MAP_L2_PROMOTION_L2_256B) ||
        !make_cand_tmap(&tvs, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p->v_self, cand_rows, cand_cols, 64, a.cpt,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B))
      return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled failed for k_self / v_self");
  }
  if (ns == 1 && make_cand_tmap(&to, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, p->out, cand_rows, cand_cols, 32, 32,
                                CU_TENSOR_MAP_L2_PROMOTION_NONE))
    a.out_tma = 1;

  // persistent grid: one CTA pair per SM pair, never more pairs than an upper bound on the item count
  const int cpb = 2 * a.cpt;
  long long max_items = ((p->total_q + cpb - 1) / cpb + p->B) * static_cast<long long>(hkv) * p->n_layers * ns;
  int pairs = sm_count() / 2;
  if (pairs <= 0) return fail(UPR_ERR_CUDA, "could not query the SM count");
  if (max_items < pairs) pairs = static_cast<int>(max_items < 1 ? 1 : max_items);
  if (p->k_self != nullptr) {
    UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::pair::upr_attn_pair_kernel<true>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, upr::pair::kSmemTotal));
    upr::pair::upr_attn_pair_kernel<true><<<2 * pairs, upr::pair::kThreads, upr::pair::kSmemTotal, st>>>(tk, tv, tq, to, tks, tvs, a);
  } else {
    UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::pair::upr_attn_pair_kernel<false>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, upr::pair::kSmemTotal));
    upr::pair::upr_attn_pair_kernel<false><<<2 * pairs, upr::pair::kThreads, upr::pair::kSmemTotal, st>>>(tk, tv, tq, to, tks, tvs, a);
  }
  UPR_CUDA_CHECK(cudaGetLastError());
  g_launches = 2;
  g_kernel = "upr_attn_pair_kernel";
  if (ns > 1) {
    s = launch_combine(a.part_o, a.part_ml, p->out, out_rows, ns, p->d, st);
    if (s != UPR_OK) return s;
    g_launches = 3;
  }
  return UPR_OK;
}

upr_status run_attn(const upr_attn_params* p, bool have_workspace, cudaStream_t st) {
  g_launches = 0;
  upr_status s = validate(p);
  if (s != UPR_OK) return s;
  if (p->B == 0 || p->total_q == 0) return UPR_OK;
  s = check_device();
  if (s != UPR_OK) return s;

  const bool pair = use_pair(p, have_workspace);
  if (p->causal && (!pair || p->num_splits > 1))
    return fail(UPR_ERR_UNSUPPORTED, "causal attention needs the CTA-pair kernel (bf16 q and K/V, d = 128, a workspace) and no split-K");
  if (p->kernel == UPR_KERNEL_PAIR && !pair)
    return fail(UPR_ERR_UNSUPPORTED, "the CTA-pair kernel needs bf16 q and K/V, d = 128, H/H_kv in {1,2,4,8}");
  const int hkv = kv_heads(p);
  if (!pair && hkv != p->H)
    return fail(UPR_ERR_UNSUPPORTED,
                "grouped queries (H_kv=%d < H=%d) need bf16 q and K/V, d = 128, H/H_kv in {2,4,8}", hkv, p->H);
  const int ns = have_workspace ? pick_splits(p, pair) : 1;
  if (have_workspace) {
    const size_t need = upr_cross_attn_workspace_bytes(p);
    if (p->workspace == nullptr || p->workspace_bytes < need)
      return fail(UPR_ERR_WORKSPACE, "workspace too small: need %zu bytes, got %zu", need,
                  p->workspace ? p->workspace_bytes : (size_t)0);
    if ((reinterpret_cast<uintptr_t>(p->workspace) & 255) != 0)
      return fail(UPR_ERR_WORKSPACE, "workspace must be 256-byte aligned");
  }
  if (pair) return run_attn_pair(p, ns, st);

  upr::AttnArgs a;
  memset(&a, 0, sizeof(a));
  a.q = p->q;
  a.k_self = p->k_self;
  a.v_self = p->v_self;
  a.out = p->out;
  a.seq_lens = p->seq_lens;
  a.cand_offsets = p->cand_offsets;
  a.k_scale = p->k_scale;
  a.v_scale = p->v_scale;
  a.B = p->B;
  a.H = p->H;
  a.n_layers = p->n_layers;
  a.num_splits = ns;
  a.q_is_f32 = (p->q_dtype == UPR_F32);
  a.scale_per_user = (p->kv_dtype == UPR_FP8_E4M3_USER);
  if (p->kv_source == UPR_KV_POOL) {
    a.slot_ids = p->slot_ids;
    a.pool_S = p->pool_slots;
    a.pool_n = p->pool_n_max;
  }
  const float sm = p->sm_scale > 0.f ? p->sm_scale : 1.0f / sqrtf(static_cast<float>(p->d));
  a.scale_log2 = sm * 1.4426950408889634f;

  const long long out_rows = static_cast<long long>(p->n_layers) * p->total_q * p->H;
  if (have_workspace) {
    a.counter = static_cast<unsigned int*>(p->workspace);
    UPR_CUDA_CHECK(cudaMemsetAsync(a.counter, 0, sizeof(unsigned int), st));
    if (ns > 1) {
      uint8_t* w = static_cast<uint8_t*>(p->workspace) + kCounterBytes + tables_bytes(p->B);
      a.part_o = reinterpret_cast<float*>(w);
      a.part_ml = a.part_o + static_cast<size_t>(out_rows) * ns * p->d;
    }
  }

  // bf16 caches are read through TMA tensor maps; fp8 / fp32 caches as contiguous raw rows
  CUtensorMap tk, tv;
  memset(&tk, 0, sizeof(tk));
  memset(&tv, 0, sizeof(tv));
  if (p->kv_dtype == UPR_BF16) {
    const long long rows = kv_view_rows(p);
    s = make_kv_tmap(&tk, p->k_cache, p->d, rows);
    if (s != UPR_OK) return s;
    s = make_kv_tmap(&tv, p->v_cache, p->d, rows);
    if (s != UPR_OK) return s;
  } else {
    if ((reinterpret_cast<uintptr_t>(p->k_cache) & 15) || (reinterpret_cast<uintptr_t>(p->v_cache) & 15))
      return fail(UPR_ERR_INVALID_ARG, "k_cache / v_cache must be 16-byte aligned");
    a.k_raw = static_cast<const uint8_t*>(p->k_cache);
    a.v_raw = static_cast<const uint8_t*>(p->v_cache);
  }

  // persistent grid: one CTA per SM, never more CTAs than an upper bound on the item count
  long long max_items = ((p->total_q + upr::kQBlock - 1) / upr::kQBlock + p->B) *
                        static_cast<long long>(p->H) * p->n_layers * ns;
  int grid = sm_count();
  if (grid <= 0) return fail(UPR_ERR_CUDA, "could not query the SM count");
  // (the plain entry point does not know total_q on the host: it always launches one CTA per SM;
  // CTAs without an item leave at once)
  if (have_workspace && max_items < grid) grid = static_cast<int>(max_items < 1 ? 1 : max_items);

  // `out` / `q` as 2-D tensors [n_layers * total_q, H * d] for the TMA stores of full tiles and the
  // TMA loads of Q tiles (need the host copy of total_q: the extended entry point only)
  CUtensorMap to, tq;
  memset(&to, 0, sizeof(to));
  memset(&tq, 0, sizeof(tq));
  const long long cand_rows = static_cast<long long>(p->n_layers) * p->total_q;
  const long long cand_cols = static_cast<long long>(p->H) * p->d;
  if (have_workspace && cand_rows < (1LL << 31)) {
    if (ns == 1 && make_cand_tmap(&to, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, p->out, cand_rows, cand_cols, 32, 32,
                                  CU_TENSOR_MAP_L2_PROMOTION_NONE))
      a.out_tma = 1;
    if (p->q_dtype == UPR_BF16 && p->kv_dtype == UPR_BF16 &&
        make_cand_tmap(&tq, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, p->q, cand_rows, cand_cols, 64, 128,
                       CU_TENSOR_MAP_L2_PROMOTION_L2_256B))
      a.q_tma = 1;
  }
  s = (p->d == 64) ? launch_attn_d<64>(p->kv_dtype, a, tk, tv, to, tq, grid, st)
                   : launch_attn_d<128>(p->kv_dtype, a, tk, tv, to, tq, grid, st);
  if (s != UPR_OK) return s;
  g_launches = 1;
  g_kernel = "upr_attn_fwd_kernel";
  if (ns > 1) {
    s = launch_combine(a.part_o, a.part_ml, p->out, out_rows, ns, p->d, st);
    if (s != UPR_OK) return s;
    g_launches = 2;
  }
  return UPR_OK;
}

}  // namespace

// ================================================================================= C ABI
extern "C" {

const char* upr_last_error(void) { return g_err; }
const char* upr_version(void) { return "upr 0.1 sm_100a"; }
int upr_last_launch_count(void) { return g_launches; }
const char* upr_last_attn_kernel(void) { return g_kernel; }

upr_status upr_kv_cache_layout(const int32_t* seq_lens, int B, int H, int d, int n_layers,
                               upr_dtype dtype, upr_kv_layout* out, int64_t* row_off) {
  if (out == nullptr) return fail(UPR_ERR_INVALID_ARG, "out is NULL");
  if (B < 0 || H <= 0 || n_layers <= 0 || d <= 0 || (B > 0 && seq_lens == nullptr))
    return fail(UPR_ERR_INVALID_ARG, "bad sizes (B=%d H=%d d=%d n_layers=%d)", B, H, d, n_layers);
  if (d != 64 && d != 128) return fail(UPR_ERR_UNSUPPORTED, "head dim d=%d unsupported", d);
  if (dtype != UPR_F32 && dtype != UPR_BF16 && dtype != UPR_FP8_E4M3 && dtype != UPR_FP8_E4M3_USER)
    return fail(UPR_ERR_UNSUPPORTED, "dtype %d unsupported", (int)dtype);
  int64_t acc = 0;
  if (row_off) row_off[0] = 0;
  for (int b = 0; b < B; ++b) {
    if (seq_lens[b] < 0) return fail(UPR_ERR_INVALID_ARG, "seq_lens[%d] = %d < 0", b, seq_lens[b]);
    acc += (static_cast<int64_t>(seq_lens[b]) + UPR_ROW_ALIGN - 1) / UPR_ROW_ALIGN * UPR_ROW_ALIGN;
    if (row_off) row_off[b + 1] = acc;
  }
  if (static_cast<int64_t>(n_layers) * H * acc + UPR_TAIL_ROWS >= (static_cast<int64_t>(1) << 31))
    return fail(UPR_ERR_UNSUPPORTED, "cache has too many rows for 32-bit TMA coordinates");
  const int eb = elem_bytes(dtype);
  out->B = B;
  out->H = H;
  out->d = d;
  out->n_layers = n_layers;
  out->dtype = dtype;
  out->row_align = UPR_ROW_ALIGN;
  out->tail_rows = UPR_TAIL_ROWS;
  out->elem_bytes = eb;
  out->R = acc;
  out->row_bytes = static_cast<int64_t>(eb) * d;
  out->head_stride_bytes = acc * eb * d;
  out->layer_stride_bytes = static_cast<int64_t>(H) * acc * eb * d;
  out->bytes_cache = (static_cast<int64_t>(n_layers) * H * acc + UPR_TAIL_ROWS) * eb * d;
  out->bytes_scales = (dtype == UPR_FP8_E4M3)        ? static_cast<int64_t>(n_layers) * H * 4
                      : (dtype == UPR_FP8_E4M3_USER) ? static_cast<int64_t>(n_layers) * B * H * 4
                                                      : 0;
  return UPR_OK;
}

upr_status upr_kv_pack(const void* k_pool, const void* v_pool, int S, int n_max,
                       const int32_t* slot_ids, const int32_t* seq_lens,
                       const upr_kv_layout* lay, void* k_cache, void* v_cache, float* k_scale,
                       float* v_scale, void* stream) {
  g_launches = 0;
  if (lay == nullptr) return fail(UPR_ERR_INVALID_ARG, "layout is NULL");
  if (S <= 0 || n_max <= 0) return fail(UPR_ERR_INVALID_ARG, "bad pool shape S=%d n_max=%d", S, n_max);
  if ((k_pool == nullptr) != (k_cache == nullptr) || (v_pool == nullptr) != (v_cache == nullptr))
    return fail(UPR_ERR_INVALID_ARG, "pool/cache pointers must be paired");
  if (lay->d != 64 && lay->d != 128) return fail(UPR_ERR_UNSUPPORTED, "d=%d unsupported", lay->d);
  if (lay->B == 0) return UPR_OK;  // nothing to gather; tail untouched
  if (slot_ids == nullptr || seq_lens == nullptr)
    return fail(UPR_ERR_INVALID_ARG, "slot_ids / seq_lens is NULL");
  const bool per_user = lay->dtype == UPR_FP8_E4M3_USER;
  const bool fp8 = lay->dtype == UPR_FP8_E4M3 || per_user;
  if (fp8 && ((k_pool && !k_scale) || (v_pool && !v_scale)))
    return fail(UPR_ERR_INVALID_ARG, "FP8 pack needs scale outputs");
  upr_status s = check_device();
  if (s != UPR_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t smem = (static_cast<size_t>(lay->B) + 1) * sizeof(int);
  if (smem > 40 * 1024) return fail(UPR_ERR_UNSUPPORTED, "B=%d too large for the pack kernel", lay->B);
  const int grid = sm_count() * 8;
  const int n_scale = lay->n_layers * lay->H * (per_user ? lay->B : 1);
  for (int which = 0; which < 2; ++which) {
    const void* pool = which == 0 ? k_pool : v_pool;
    if (pool == nullptr) continue;
    upr::PackArgs a;
    a.pool = static_cast<const __nv_bfloat16*>(pool);
    a.cache = which == 0 ? k_cache : v_cache;
    a.scale = which == 0 ? k_scale : v_scale;
    a.slot_ids = slot_ids;
    a.seq_lens = seq_lens;
    a.B = lay->B;
    a.H = lay->H;
    a.d = lay->d;
    a.n_layers = lay->n_layers;
    a.S = S;
    a.n_max = n_max;
    a.tail_rows = lay->tail_rows;
    a.per_user = per_user ? 1 : 0;
    const bool d64 = lay->d == 64;
#define UPR_PACK_LAUNCH(MODE)                                                              \
  do {                                                                                     \
    if (d64) upr::upr_pack_kernel<MODE, 64><<<grid, upr::kPackThreads, smem, st>>>(a);     \
    else upr::upr_pack_kernel<MODE, 128><<<grid, upr::kPackThreads, smem, st>>>(a);        \
  } while (0)
    if (lay->dtype == UPR_BF16) {
      UPR_PACK_LAUNCH(0);
      g_launches += 1;
    } else if (lay->dtype == UPR_F32) {
      UPR_PACK_LAUNCH(2);
      g_launches += 1;
    } else {
      UPR_CUDA_CHECK(cudaMemsetAsync(a.scale, 0, n_scale * sizeof(float), st));
      UPR_PACK_LAUNCH(3);
      UPR_PACK_LAUNCH(1);
      upr::upr_scale_finalize_kernel<<<(n_scale + 127) / 128, 128, 0, st>>>(a.scale, n_scale);
      g_launches += 3;
    }
#undef UPR_PACK_LAUNCH
    UPR_CUDA_CHECK(cudaGetLastError());
  }
  return UPR_OK;
}

namespace {
// Workspaces the library owns for the plain entry point: one per (device, stream), grown on demand, kept
// until the library is unloaded.  Calls on one stream are ordered, so they may share the scheduler state.
struct OwnedWs { int device; cudaStream_t stream; void* ptr; size_t bytes; };
std::mutex g_ws_mutex;
std::vector<OwnedWs> g_ws;

upr_status owned_workspace(cudaStream_t st, size_t need, void** out) {
  int dev = 0;
  UPR_CUDA_CHECK(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_ws_mutex);
  OwnedWs* slot = nullptr;
  for (auto& w : g_ws)
    if (w.device == dev && w.stream == st) slot = &w;
  if (slot == nullptr) {
    g_ws.push_back({dev, st, nullptr, 0});
    slot = &g_ws.back();
  }
  if (slot->bytes < need) {
    if (slot->ptr != nullptr) {
      UPR_CUDA_CHECK(cudaStreamSynchronize(st));   // an earlier call on this stream may still use it
      UPR_CUDA_CHECK(cudaFree(slot->ptr));
      slot->ptr = nullptr;
      slot->bytes = 0;
    }
    const size_t bytes = (need + (1u << 20) - 1) >> 20 << 20;
    UPR_CUDA_CHECK(cudaMalloc(&slot->ptr, bytes));
    slot->bytes = bytes;
  }
  *out = slot->ptr;
  return UPR_OK;
}
}  // namespace

upr_status upr_cross_attn_fwd(const void* q, const void* k_cache, const void* v_cache,
                              const int32_t* seq_lens, const int32_t* cand_offsets, float* out,
                              int B, int H, int d, upr_dtype dtype, void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  upr_attn_params p;
  memset(&p, 0, sizeof(p));
  p.q = q;
  p.k_cache = k_cache;
  p.v_cache = v_cache;
  p.seq_lens = seq_lens;
  p.cand_offsets = cand_offsets;
  p.out = out;
  p.B = B;
  p.H = H;
  p.d = d;
  p.n_layers = 1;
  p.kv_dtype = dtype;
  p.q_dtype = (dtype == UPR_F32) ? UPR_F32 : UPR_BF16;
  p.num_splits = 1;
  if (B <= 0 || cand_offsets == nullptr) {
    p.total_q = (B == 0) ? 0 : 1;
    return run_attn(&p, /*have_workspace=*/false, st);   // B == 0: no launch; otherwise validate() reports it
  }
  // The same path upr_cross_attn_fwd_ex takes (device-built longest-first work list, dynamic scheduler, TMA
  // q / out tiles, the CTA-pair kernel where it applies) needs the number of query rows on the host and a
  // workspace: ΣC = cand_offsets[B] is read back (4 bytes, one stream synchronisation) and the library
  // supplies the workspace.  While the stream is being captured into a CUDA graph no read-back is possible:
  // the call then runs the static schedule of the 1-CTA kernel, which needs neither.
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  UPR_CUDA_CHECK(cudaStreamIsCapturing(st, &cap));
  if (cap != cudaStreamCaptureStatusNone) {
    p.total_q = 1;   // unknown on the host; only used to skip empty launches
    return run_attn(&p, /*have_workspace=*/false, st);
  }
  int32_t total_q = 0;
  UPR_CUDA_CHECK(cudaMemcpyAsync(&total_q, cand_offsets + B, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  UPR_CUDA_CHECK(cudaStreamSynchronize(st));
  if (total_q < 0) return fail(UPR_ERR_INVALID_ARG, "cand_offsets[B] = %d is negative", (int)total_q);
  p.total_q = total_q;
  if (total_q == 0) return run_attn(&p, /*have_workspace=*/false, st);
  const size_t need = upr_cross_attn_workspace_bytes(&p);
  void* ws = nullptr;
  upr_status s = owned_workspace(st, need, &ws);
  if (s != UPR_OK) return s;
  p.workspace = ws;
  p.workspace_bytes = need;
  return run_attn(&p, /*have_workspace=*/true, st);
}

int upr_cross_attn_num_splits(const upr_attn_params* p) {
  if (p == nullptr || p->H <= 0 || (p->H_kv > 0 && p->H % p->H_kv != 0)) return 1;
  return pick_splits(p, use_pair(p, true));
}

size_t upr_cross_attn_workspace_bytes(const upr_attn_params* p) {
  if (p == nullptr || p->B < 0 || p->H <= 0 || p->n_layers <= 0 || p->total_q < 0 ||
      (p->d != 64 && p->d != 128) || (p->H_kv > 0 && p->H % p->H_kv != 0))
    return 0;
  const int ns = pick_splits(p, use_pair(p, true));
  size_t bytes = kCounterBytes + tables_bytes(p->B);
  if (ns > 1) {
    const size_t rows = static_cast<size_t>(p->n_layers) * p->total_q * p->H;
    bytes += rows * ns * (static_cast<size_t>(p->d) + 2) * sizeof(float);
  }
  return bytes;
}

upr_status upr_cross_attn_fwd_ex(const upr_attn_params* p, void* stream) {
  return run_attn(p, /*have_workspace=*/true, static_cast<cudaStream_t>(stream));
}

// ------------------------------------------------------------------ the entry point that allocates nothing
// Scratch of upr_cross_attn_fwd_noalloc: the workspace of upr_cross_attn_fwd_ex (scheduler counter, work-list
// tables, split-K partials) as a file-scope device array.  Every GPU that loads the library holds these bytes until
// the process exits.  In HOST code `g_noalloc_scratch` is only a stand-in for the symbol, not a device address: the
// address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_noalloc_scratch[UPR_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_noalloc_mutex;
void* g_noalloc_ptr[kMaxDevices] = {};   // device address of g_noalloc_scratch on device i, or nullptr = not asked yet

upr_status noalloc_scratch(void** out) {
  int dev = 0;
  UPR_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(UPR_ERR_UNSUPPORTED, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (g_noalloc_ptr[dev] == nullptr) {
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);   // device `dev` is current
    if (e != cudaSuccess || ptr == nullptr)
      return fail(UPR_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch) on device %d: %s", dev, cudaGetErrorString(e));
    if ((reinterpret_cast<uintptr_t>(ptr) & 255) != 0)
      return fail(UPR_ERR_CUDA, "static scratch is not 256-byte aligned");
    g_noalloc_ptr[dev] = ptr;
  }
  *out = g_noalloc_ptr[dev];
  return UPR_OK;
}
}  // namespace

size_t upr_cross_attn_noalloc_scratch_bytes(void) { return UPR_NOALLOC_SCRATCH_BYTES; }

upr_status upr_cross_attn_fwd_noalloc(const upr_attn_params* p, void* stream) {
  g_launches = 0;
  if (p == nullptr) return fail(UPR_ERR_INVALID_ARG, "params is NULL");
  upr_attn_params q = *p;
  q.workspace = nullptr;
  q.workspace_bytes = 0;
  const size_t need = upr_cross_attn_workspace_bytes(&q);
  if (need == 0) return run_attn(&q, /*have_workspace=*/true, static_cast<cudaStream_t>(stream));   // invalid sizes: validate() names them
  if (need > static_cast<size_t>(UPR_NOALLOC_SCRATCH_BYTES))
    return fail(UPR_ERR_WORKSPACE,
                "upr_cross_attn_fwd_noalloc: this call needs %zu bytes of scratch, the static scratch holds %zu "
                "(UPR_NOALLOC_SCRATCH_BYTES); lower num_splits / total_q, or use upr_cross_attn_fwd_ex with a workspace",
                need, static_cast<size_t>(UPR_NOALLOC_SCRATCH_BYTES));
  if (q.B == 0 || q.total_q == 0) return run_attn(&q, /*have_workspace=*/false, static_cast<cudaStream_t>(stream));
  void* ws = nullptr;
  upr_status s = noalloc_scratch(&ws);
  if (s != UPR_OK) return s;
  q.workspace = ws;
  q.workspace_bytes = UPR_NOALLOC_SCRATCH_BYTES;
  // everything in the scratch that must start from a known state is written by the call itself before it is read:
  // the scheduler counter and the work-list tables by the schedule kernel / a memset, every split-K partial the
  // combine kernel reads by the attention kernel.  Nothing of an earlier call's contents is used.
  return run_attn(&q, /*have_workspace=*/true, static_cast<cudaStream_t>(stream));
}

// ------------------------------------------------------------------ decode-layer tail, consumer, pool
namespace {
struct KvScatter { const int32_t* tok_slot; const int32_t* tok_pos; int layer, S, H, n, d; const void* residual;
                   int fp8; float x_scale, w_scale; float y_scale = 1.f; };
}  // namespace

static upr_status linear_impl(const void* x, upr_dtype x_dtype, const void* w, const float* bias, void* y,
                              upr_dtype y_dtype, int64_t M, int N, int K, upr_activation act, const KvScatter* kv,
                              void* stream) {
  g_launches = 0;
  if (M < 0 || N <= 0 || K <= 0) return fail(UPR_ERR_INVALID_ARG, "bad sizes M=%lld N=%d K=%d", (long long)M, N, K);
  const bool fp8 = kv != nullptr && kv->fp8;
  const bool xq = fp8 && x_dtype == UPR_FP8_E4M3;   // x already e4m3 in memory
  const bool yq = fp8 && y_dtype == UPR_FP8_E4M3;   // y leaves as e4m3
  if (x_dtype != UPR_BF16 && x_dtype != UPR_F32 && !xq)
    return fail(UPR_ERR_UNSUPPORTED, "x_dtype %d (bf16 or f32; e4m3 for FP8 layers)", (int)x_dtype);
  if (y_dtype != UPR_BF16 && y_dtype != UPR_F32 && !yq)
    return fail(UPR_ERR_UNSUPPORTED, "y_dtype %d (bf16 or f32; e4m3 for FP8 layers)", (int)y_dtype);
  if (act != UPR_ACT_NONE && act != UPR_ACT_SILU && act != UPR_ACT_RELU)
    return fail(UPR_ERR_INVALID_ARG, "activation %d unknown", (int)act);
  if (K % (fp8 ? 128 : 64) != 0 || N % 8 != 0)
    return fail(UPR_ERR_UNSUPPORTED, "K=%d must be a multiple of %d, N=%d of 8", K, fp8 ? 128 : 64, N);
  if (fp8 && x_dtype == UPR_F32) return fail(UPR_ERR_UNSUPPORTED, "FP8 linear layers take bf16 or e4m3 activations");
  if (fp8 && (!(kv->x_scale > 0.f) || !(kv->w_scale > 0.f) || (yq && !(kv->y_scale > 0.f))))
    return fail(UPR_ERR_INVALID_ARG, "scales must be > 0");
  if (M == 0) return UPR_OK;
  if (!x || !w || !y) return fail(UPR_ERR_INVALID_ARG, "NULL tensor pointer");
  if ((reinterpret_cast<uintptr_t>(x) & 15) || (reinterpret_cast<uintptr_t>(w) & 15) || (reinterpret_cast<uintptr_t>(y) & 15))
    return fail(UPR_ERR_INVALID_ARG, "x, w, y must be 16-byte aligned");
  if (M >= (1LL << 31)) return fail(UPR_ERR_UNSUPPORTED, "M too large for 32-bit TMA coordinates");
  upr_status s = check_device();
  if (s != UPR_OK) return s;
  EncodeTiledFn enc = get_encode_fn();
  if (enc == nullptr) return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
  CUtensorMap tx, tw;
  cuuint32_t box[2] = {static_cast<cuuint32_t>(fp8 ? 128 : 64), 128}, estr[2] = {1, 1};
  {
    const bool f32 = x_dtype == UPR_F32;
    cuuint64_t gdim[2] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(M)};
    cuuint64_t gstride[1] = {static_cast<cuuint64_t>(K) * (f32 ? 4 : xq ? 1 : 2)};
    if (enc(&tx, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : xq ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
            2, const_cast<void*>(x),
            gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            (f32 || (fp8 && !xq)) ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled failed for x");
  }
  {
    cuuint64_t gdim[2] = {static_cast<cuuint64_t>(K), static_cast<cuuint64_t>(N)};
    cuuint64_t gstride[1] = {static_cast<cuuint64_t>(K) * (fp8 ? 1 : 2)};
    if (enc(&tw, fp8 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(w), gdim,
            gstride, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled failed for w");
  }
  upr::lin::Args a;
  memset(&a, 0, sizeof(a));
  if (kv != nullptr) a.residual = static_cast<const __nv_bfloat16*>(kv->residual);
  if (kv != nullptr && kv->tok_slot != nullptr) {
    a.tok_slot = kv->tok_slot;
    a.tok_pos = kv->tok_pos;
    a.kv_layer = kv->layer;
    a.kv_S = kv->S;
    a.kv_H = kv->H;
    a.kv_n = kv->n;
    a.kv_d = kv->d;
  }
  a.bias = bias;
  a.y = y;
  a.M = M;
  a.N = N;
  a.K = K;
  a.act = static_cast<int>(act);
  a.y_is_f32 = y_dtype == UPR_F32;
  a.out_scale = fp8 ? kv->x_scale * kv->w_scale : 1.0f;
  a.x_mult = fp8 ? 1.0f / kv->x_scale : 1.0f;
  a.y_is_fp8 = yq ? 1 : 0;
  a.y_mult = yq ? 1.0f / kv->y_scale : 1.0f;
  int sms = sm_count();
  if (sms <= 0) return fail(UPR_ERR_CUDA, "could not query the SM count");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // 256 x 256 tiles on CTA pairs when there are enough of them to fill the machine's SM pairs; small problems
  // (and narrow layers, N <= 128) keep the 128 x 128 single-CTA kernel
  const long long tiles2 = ((M + 255) / 256) * ((N + 255) / 256);
  if (fp8 || (N > 128 && tiles2 >= sms / 2)) {
    int pairs = sms / 2;
    if (tiles2 < pairs) pairs = static_cast<int>(tiles2);
    if (xq) {
      using C = upr::lin2::Cfg<upr::lin2::MODE_FP8Q>;
      UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_FP8Q>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemTotal));
      upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_FP8Q><<<2 * pairs, upr::lin2::kThreads, C::kSmemTotal, st>>>(tx, tw, a);
    } else if (fp8) {
      using C = upr::lin2::Cfg<upr::lin2::MODE_FP8>;
      UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_FP8>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemTotal));
      upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_FP8><<<2 * pairs, upr::lin2::kThreads, C::kSmemTotal, st>>>(tx, tw, a);
    } else if (x_dtype == UPR_F32) {
      using C = upr::lin2::Cfg<upr::lin2::MODE_XF32>;
      UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_XF32>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemTotal));
      upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_XF32><<<2 * pairs, upr::lin2::kThreads, C::kSmemTotal, st>>>(tx, tw, a);
    } else {
      using C = upr::lin2::Cfg<upr::lin2::MODE_BF16>;
      UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_BF16>,
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, C::kSmemTotal));
      upr::lin2::upr_linear_pair_kernel<upr::lin2::MODE_BF16><<<2 * pairs, upr::lin2::kThreads, C::kSmemTotal, st>>>(tx, tw, a);
    }
    UPR_CUDA_CHECK(cudaGetLastError());
    g_launches = 1;
    return UPR_OK;
  }
  const long long tiles = ((M + 127) / 128) * ((N + 127) / 128);
  int grid = sms;
  if (tiles < grid) grid = static_cast<int>(tiles);
  if (x_dtype == UPR_F32) {
    UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::lin::upr_linear_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        upr::lin::kSmemTotal));
    upr::lin::upr_linear_kernel<true><<<grid, upr::lin::kThreads, upr::lin::kSmemTotal, st>>>(tx, tw, a);
  } else {
    UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::lin::upr_linear_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        upr::lin::kSmemTotal));
    upr::lin::upr_linear_kernel<false><<<grid, upr::lin::kThreads, upr::lin::kSmemTotal, st>>>(tx, tw, a);
  }
  UPR_CUDA_CHECK(cudaGetLastError());
  g_launches = 1;
  return UPR_OK;
}

upr_status upr_linear_fwd(const void* x, upr_dtype x_dtype, const void* w, const float* bias, void* y,
                          upr_dtype y_dtype, int64_t M, int N, int K, upr_activation act, void* stream) {
  return linear_impl(x, x_dtype, w, bias, y, y_dtype, M, N, K, act, nullptr, stream);
}

upr_status upr_linear_residual_fwd(const void* x, upr_dtype x_dtype, const void* w, const float* bias,
                                   const void* residual, void* y, upr_dtype y_dtype, int64_t M, int N, int K,
                                   upr_activation act, void* stream) {
  if (residual != nullptr && (reinterpret_cast<uintptr_t>(residual) & 15))
    return fail(UPR_ERR_INVALID_ARG, "residual must be 16-byte aligned");
  KvScatter kv{nullptr, nullptr, 0, 0, 0, 0, 0, residual, 0, 1.f, 1.f};
  return linear_impl(x, x_dtype, w, bias, y, y_dtype, M, N, K, act, &kv, stream);
}

upr_status upr_linear_fp8_fwd(const void* x, float x_scale, const void* w_e4m3, float w_scale, const float* bias,
                              const void* residual, void* y, upr_dtype y_dtype, int64_t M, int N, int K,
                              upr_activation act, void* stream) {
  if (residual != nullptr && (reinterpret_cast<uintptr_t>(residual) & 15))
    return fail(UPR_ERR_INVALID_ARG, "residual must be 16-byte aligned");
  KvScatter kv{nullptr, nullptr, 0, 0, 0, 0, 0, residual, 1, x_scale, w_scale};
  return linear_impl(x, UPR_BF16, w_e4m3, bias, y, y_dtype, M, N, K, act, &kv, stream);
}

upr_status upr_linear_fp8_ex_fwd(const void* x, upr_dtype x_dtype, float x_scale, const void* w_e4m3, float w_scale,
                                 const float* bias, const void* residual, void* y, upr_dtype y_dtype, float y_scale,
                                 int64_t M, int N, int K, upr_activation act, void* stream) {
  if (residual != nullptr && (reinterpret_cast<uintptr_t>(residual) & 15))
    return fail(UPR_ERR_INVALID_ARG, "residual must be 16-byte aligned");
  if (x_dtype != UPR_BF16 && x_dtype != UPR_FP8_E4M3)
    return fail(UPR_ERR_UNSUPPORTED, "x_dtype %d (bf16 or e4m3)", (int)x_dtype);
  KvScatter kv{nullptr, nullptr, 0, 0, 0, 0, 0, residual, 1, x_scale, w_scale, y_scale};
  return linear_impl(x, x_dtype, w_e4m3, bias, y, y_dtype, M, N, K, act, &kv, stream);
}

static upr_status layernorm_impl(const void* x, const float* gamma, const float* beta, void* y, bool y_fp8, float y_scale,
                                 int64_t M, int D, float eps, void* stream) {
  g_launches = 0;
  if (M < 0 || D <= 0) return fail(UPR_ERR_INVALID_ARG, "bad sizes M=%lld D=%d", (long long)M, D);
  if (D % 8 != 0 || D > 4096) return fail(UPR_ERR_UNSUPPORTED, "D=%d must be a multiple of 8 and <= 4096", D);
  if (y_fp8 && !(y_scale > 0.f)) return fail(UPR_ERR_INVALID_ARG, "y_scale must be > 0");
  if (M == 0) return UPR_OK;
  if (!x || !gamma || !beta || !y) return fail(UPR_ERR_INVALID_ARG, "NULL tensor pointer");
  upr_status s = check_device();
  if (s != UPR_OK) return s;
  const long long blocks = (M + 7) / 8;
  const int grid = static_cast<int>(blocks < sm_count() * 8LL ? blocks : sm_count() * 8LL);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (y_fp8)
    upr::upr_layernorm_kernel<true><<<grid, 256, 0, st>>>(static_cast<const __nv_bfloat16*>(x), gamma, beta, M, D, eps, y,
                                                          1.0f / y_scale);
  else
    upr::upr_layernorm_kernel<false><<<grid, 256, 0, st>>>(static_cast<const __nv_bfloat16*>(x), gamma, beta, M, D, eps, y,
                                                           1.0f);
  UPR_CUDA_CHECK(cudaGetLastError());
  g_launches = 1;
  return UPR_OK;
}

upr_status upr_layernorm_fwd(const void* x, const float* gamma, const float* beta, void* y, int64_t M, int D,
                             float eps, void* stream) {
  return layernorm_impl(x, gamma, beta, y, false, 1.f, M, D, eps, stream);
}

upr_status upr_layernorm_fp8_fwd(const void* x, const float* gamma, const float* beta, void* y_e4m3, float y_scale,
                                 int64_t M, int D, float eps, void* stream) {
  return layernorm_impl(x, gamma, beta, y_e4m3, true, y_scale, M, D, eps, stream);
}

upr_status upr_kv_project_into_pool(const void* x, upr_dtype x_dtype, const void* w, const float* bias, void* pool,
                                    const int32_t* tok_slot, const int32_t* tok_pos, int64_t M, int K, int layer,
                                    int n_layers, int S, int H, int n, int d, void* stream) {
  if (S <= 0 || H <= 0 || n <= 0 || n_layers <= 0 || layer < 0 || layer >= n_layers)
    return fail(UPR_ERR_INVALID_ARG, "bad pool shape / layer (layers=%d S=%d H=%d n=%d layer=%d)", n_layers, S, H, n, layer);
  if (d != 64 && d != 128) return fail(UPR_ERR_UNSUPPORTED, "head dim d=%d unsupported (64 or 128)", d);
  if (M > 0 && (!tok_slot || !tok_pos)) return fail(UPR_ERR_INVALID_ARG, "tok_slot / tok_pos is NULL");
  KvScatter kv{tok_slot, tok_pos, layer, S, H, n, d, nullptr, 0, 1.f, 1.f};
  return linear_impl(x, x_dtype, w, bias, pool, UPR_BF16, M, H * d, K, UPR_ACT_NONE, &kv, stream);
}

upr_status upr_action_utility(const void* hid, const float* w2, const float* b2, const float* wc, int64_t M,
                              int C, int Dh, float* probs, float* util, void* stream) {
  g_launches = 0;
  if (M < 0 || C <= 0 || Dh <= 0) return fail(UPR_ERR_INVALID_ARG, "bad sizes M=%lld C=%d Dh=%d", (long long)M, C, Dh);
  if (Dh % 8 != 0) return fail(UPR_ERR_UNSUPPORTED, "Dh=%d must be a multiple of 8", Dh);
  if (M == 0) return UPR_OK;
  if (!hid || !w2 || !b2 || !wc || !util) return fail(UPR_ERR_INVALID_ARG, "NULL tensor pointer");
  upr_status s = check_device();
  if (s != UPR_OK) return s;
  const long long blocks = (M + 7) / 8;
  const int grid = static_cast<int>(blocks < sm_count() * 8LL ? blocks : sm_count() * 8LL);
  upr::upr_head_utility_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(
      static_cast<const __nv_bfloat16*>(hid), w2, b2, wc, M, C, Dh, probs, util);
  UPR_CUDA_CHECK(cudaGetLastError());
  g_launches = 1;
  return UPR_OK;
}

upr_status upr_topk_per_user(const float* util, const int32_t* cand_offsets, int B, int K, int max_cands,
                             int32_t* out_idx, int32_t* out_cnt, void* stream) {
  g_launches = 0;
  if (B < 0 || K <= 0 || max_cands < 0) return fail(UPR_ERR_INVALID_ARG, "bad sizes B=%d K=%d max_cands=%d", B, K, max_cands);
  if (max_cands > 16384) return fail(UPR_ERR_UNSUPPORTED, "max_cands=%d > 16384 candidates per user", max_cands);
  if (B == 0) return UPR_OK;
  if (!util || !cand_offsets || !out_idx || !out_cnt) return fail(UPR_ERR_INVALID_ARG, "NULL tensor pointer");
  upr_status s = check_device();
  if (s != UPR_OK) return s;
  int n_pad = 2;
  while (n_pad < max_cands) n_pad <<= 1;
  const size_t smem = static_cast<size_t>(n_pad) * sizeof(unsigned long long);
  UPR_CUDA_CHECK(cudaFuncSetAttribute(upr::upr_topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      static_cast<int>(smem)));
  upr::upr_topk_kernel<<<B, upr::kTopkThreads, smem, static_cast<cudaStream_t>(stream)>>>(util, cand_offsets, K, n_pad,
                                                                                            out_idx, out_cnt);
  UPR_CUDA_CHECK(cudaGetLastError());
  g_launches = 1;
  return UPR_OK;
}

static_assert(sizeof(cudaIpcMemHandle_t) + 8 <= UPR_IPC_HANDLE_BYTES, "IPC handle does not fit");

typedef CUresult (*GetAddressRangeFn)(CUdeviceptr*, size_t*, CUdeviceptr);

upr_status upr_pool_export(const void* pool_dev, upr_ipc_handle* out) {
  if (!pool_dev || !out) return fail(UPR_ERR_INVALID_ARG, "NULL argument");
  void* fnp = nullptr;
  cudaDriverEntryPointQueryResult qres;
  UPR_CUDA_CHECK(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fnp, cudaEnableDefault, &qres));
  if (fnp == nullptr || qres != cudaDriverEntryPointSuccess)
    return fail(UPR_ERR_CUDA, "cuMemGetAddressRange entry point not found");
  CUdeviceptr base = 0;
  size_t size = 0;
  if (reinterpret_cast<GetAddressRangeFn>(fnp)(&base, &size, reinterpret_cast<CUdeviceptr>(pool_dev)) != CUDA_SUCCESS)
    return fail(UPR_ERR_INVALID_ARG, "pool_dev is not inside a device allocation of this process");
  cudaIpcMemHandle_t h;
  UPR_CUDA_CHECK(cudaIpcGetMemHandle(&h, reinterpret_cast<void*>(base)));
  const uint64_t offset = reinterpret_cast<CUdeviceptr>(pool_dev) - base;
  memset(out->bytes, 0, sizeof(out->bytes));
  memcpy(out->bytes, &h, sizeof(h));
  memcpy(out->bytes + sizeof(h), &offset, sizeof(offset));
  return UPR_OK;
}

namespace {
// open mappings of this process: translated pointer -> mapped base (upr_pool_close needs the base)
struct OpenPool { void* ptr; void* base; };
OpenPool g_open[64];
int g_n_open = 0;
}  // namespace

upr_status upr_pool_open(const upr_ipc_handle* handle, void** pool_dev) {
  if (!handle || !pool_dev) return fail(UPR_ERR_INVALID_ARG, "NULL argument");
  if (g_n_open >= 64) return fail(UPR_ERR_UNSUPPORTED, "too many open pools");
  cudaIpcMemHandle_t h;
  uint64_t offset = 0;
  memcpy(&h, handle->bytes, sizeof(h));
  memcpy(&offset, handle->bytes + sizeof(h), sizeof(offset));
  void* base = nullptr;
  UPR_CUDA_CHECK(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
  *pool_dev = static_cast<uint8_t*>(base) + offset;
  g_open[g_n_open++] = OpenPool{*pool_dev, base};
  return UPR_OK;
}

upr_status upr_pool_close(void* pool_dev) {
  if (!pool_dev) return fail(UPR_ERR_INVALID_ARG, "NULL argument");
  for (int i = 0; i < g_n_open; ++i)
    if (g_open[i].ptr == pool_dev) {
      void* base = g_open[i].base;
      g_open[i] = g_open[--g_n_open];
      UPR_CUDA_CHECK(cudaIpcCloseMemHandle(base));
      return UPR_OK;
    }
  return fail(UPR_ERR_INVALID_ARG, "pointer was not returned by upr_pool_open");
}

upr_status upr_slot_ring_init(upr_slot_ring* ring, int32_t S) {
  if (!ring || S <= 0) return fail(UPR_ERR_INVALID_ARG, "bad slot ring (S=%d)", S);
  ring->S = S;
  ring->next = 0;
  return UPR_OK;
}

upr_status upr_slot_ring_acquire(upr_slot_ring* ring, int32_t n, int32_t* slot_ids_host) {
  if (!ring || ring->S <= 0 || n < 0 || (n > 0 && !slot_ids_host)) return fail(UPR_ERR_INVALID_ARG, "bad slot ring request");
  if (n > ring->S) return fail(UPR_ERR_INVALID_ARG, "%d slots requested from a pool of %d: a batch would overwrite itself", n, ring->S);
  for (int32_t i = 0; i < n; ++i) {
    slot_ids_host[i] = ring->next;
    ring->next = (ring->next + 1) % ring->S;
  }
  return UPR_OK;
}

}  // extern "C"
