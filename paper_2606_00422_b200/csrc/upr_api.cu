// upr_api.cu -- C ABI of libupr (include/upr.h): argument checks, tensor-map encoding, launches.
// No torch types, no host synchronisation, no device allocation.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <atomic>

#include "../../include/upr.h"
#include "attn_kernel.cuh"
#include "pack_kernels.cuh"

namespace {

thread_local char g_err[512] = "";
thread_local int g_launches = 0;

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

// 2-D bf16 view [rows, d] of a packed cache; box = [128 rows x 64 cols], 128-byte swizzle.
// The row extent is left unbounded (the layout contract guarantees UPR_TAIL_ROWS of slack),
// because R depends on device-resident seq_lens the host never reads.
upr_status make_kv_tmap(CUtensorMap* m, const void* base, int d) {
  EncodeTiledFn enc = get_encode_fn();
  if (enc == nullptr) return fail(UPR_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t gdim[2] = {static_cast<cuuint64_t>(d), static_cast<cuuint64_t>(1) << 31};
  cuuint64_t gstride[1] = {static_cast<cuuint64_t>(d) * 2};
  cuuint32_t box[2] = {64, 128};
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

int pick_splits(const upr_attn_params* p) {
  if (p->num_splits >= 1) return p->num_splits;
  // heuristic: split the history when the (user, head, q-block) items cannot fill the SMs
  if (p->max_seq_len <= 0 || p->total_q <= 0 || p->B <= 0) return 1;
  const int sms = sm_count() > 0 ? sm_count() : 148;
  const long long blocks = (p->total_q + upr::kQBlock - 1) / upr::kQBlock + p->B / 2;
  const long long items = blocks * p->H * p->n_layers;
  const int tiles = (p->max_seq_len + upr::kTileN - 1) / upr::kTileN;
  if (items >= 2LL * sms || tiles < 4) return 1;
  long long want = (2LL * sms + items - 1) / items;
  long long cap = tiles / 2;  // at least two tiles per split
  long long ns = want < cap ? want : cap;
  if (ns > 16) ns = 16;
  return ns < 1 ? 1 : static_cast<int>(ns);
}

upr_status validate(const upr_attn_params* p) {
  if (p == nullptr) return fail(UPR_ERR_INVALID_ARG, "params is NULL");
  if (p->B < 0 || p->H <= 0 || p->n_layers <= 0 || p->total_q < 0)
    return fail(UPR_ERR_INVALID_ARG, "negative or zero size (B=%d H=%d n_layers=%d total_q=%lld)",
                p->B, p->H, p->n_layers, (long long)p->total_q);
  if (p->d != 64 && p->d != 128)
    return fail(UPR_ERR_UNSUPPORTED, "head dim d=%d unsupported (64 or 128)", p->d);
  if (p->kv_dtype != UPR_BF16 && p->kv_dtype != UPR_FP8_E4M3 && p->kv_dtype != UPR_F32)
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
    case UPR_FP8_E4M3: return launch_attn<D, upr::KV_FP8>(a, tk, tv, to, tq, grid, st);
    default: return launch_attn<D, upr::KV_F32>(a, tk, tv, to, tq, grid, st);
  }
}

upr_status run_attn(const upr_attn_params* p, bool have_workspace, cudaStream_t st) {
  g_launches = 0;
  upr_status s = validate(p);
  if (s != UPR_OK) return s;
  if (p->B == 0 || p->total_q == 0) return UPR_OK;
  s = check_device();
  if (s != UPR_OK) return s;

  const int ns = have_workspace ? pick_splits(p) : 1;
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
  const float sm = p->sm_scale > 0.f ? p->sm_scale : 1.0f / sqrtf(static_cast<float>(p->d));
  a.scale_log2 = sm * 1.4426950408889634f;

  const long long out_rows = static_cast<long long>(p->n_layers) * p->total_q * p->H;
  if (have_workspace) {
    const size_t need = upr_cross_attn_workspace_bytes(p);
    if (p->workspace == nullptr || p->workspace_bytes < need)
      return fail(UPR_ERR_WORKSPACE, "workspace too small: need %zu bytes, got %zu", need,
                  p->workspace ? p->workspace_bytes : (size_t)0);
    if ((reinterpret_cast<uintptr_t>(p->workspace) & 255) != 0)
      return fail(UPR_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    a.counter = static_cast<unsigned int*>(p->workspace);
    UPR_CUDA_CHECK(cudaMemsetAsync(a.counter, 0, sizeof(unsigned int), st));
    if (ns > 1) {
      uint8_t* w = static_cast<uint8_t*>(p->workspace) + kCounterBytes;
      a.part_o = reinterpret_cast<float*>(w);
      a.part_ml = a.part_o + static_cast<size_t>(out_rows) * ns * p->d;
    }
  }

  // bf16 caches are read through TMA tensor maps; fp8 / fp32 caches as contiguous raw rows
  CUtensorMap tk, tv;
  memset(&tk, 0, sizeof(tk));
  memset(&tv, 0, sizeof(tv));
  if (p->kv_dtype == UPR_BF16) {
    s = make_kv_tmap(&tk, p->k_cache, p->d);
    if (s != UPR_OK) return s;
    s = make_kv_tmap(&tv, p->v_cache, p->d);
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

  // `out` as a 2-D fp32 tensor [n_layers * total_q, H * d] for the TMA stores of full tiles
  // (needs the host copy of total_q: the extended entry point only)
  CUtensorMap to;
  memset(&to, 0, sizeof(to));
  if (have_workspace && ns == 1 && p->total_q > 0 &&
      static_cast<long long>(p->n_layers) * p->total_q < (1LL << 31)) {
    EncodeTiledFn enc = get_encode_fn();
    cuuint64_t gdim[2] = {static_cast<cuuint64_t>(p->H) * p->d,
                          static_cast<cuuint64_t>(p->n_layers) * static_cast<cuuint64_t>(p->total_q)};
    cuuint64_t gstride[1] = {static_cast<cuuint64_t>(p->H) * p->d * sizeof(float)};
    cuuint32_t box[2] = {32, 32};
    cuuint32_t estr[2] = {1, 1};
    if (enc != nullptr &&
        enc(&to, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, p->out, gdim, gstride, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS)
      a.out_tma = 1;
  }
  // `q` as a 2-D bf16 tensor [n_layers * total_q, H * d]: Q tiles by TMA (bf16 q and cache only)
  CUtensorMap tq;
  memset(&tq, 0, sizeof(tq));
  if (have_workspace && p->total_q > 0 && p->q_dtype == UPR_BF16 && p->kv_dtype == UPR_BF16 &&
      static_cast<long long>(p->n_layers) * p->total_q < (1LL << 31)) {
    EncodeTiledFn enc = get_encode_fn();
    cuuint64_t gdim[2] = {static_cast<cuuint64_t>(p->H) * p->d,
                          static_cast<cuuint64_t>(p->n_layers) * static_cast<cuuint64_t>(p->total_q)};
    cuuint64_t gstride[1] = {static_cast<cuuint64_t>(p->H) * p->d * 2};
    cuuint32_t box[2] = {64, 128};
    cuuint32_t estr[2] = {1, 1};
    if (enc != nullptr &&
        enc(&tq, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(p->q), gdim, gstride, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS)
      a.q_tma = 1;
  }
  s = (p->d == 64) ? launch_attn_d<64>(p->kv_dtype, a, tk, tv, to, tq, grid, st)
                   : launch_attn_d<128>(p->kv_dtype, a, tk, tv, to, tq, grid, st);
  if (s != UPR_OK) return s;
  g_launches = 1;
  if (ns > 1) {
    long long blocks = (out_rows + 7) / 8;
    int cgrid = static_cast<int>(blocks < sm_count() * 8LL ? blocks : sm_count() * 8LL);
    if (p->d == 64)
      upr::upr_combine_kernel<64><<<cgrid, 256, 0, st>>>(a.part_o, a.part_ml, p->out, out_rows, ns);
    else
      upr::upr_combine_kernel<128><<<cgrid, 256, 0, st>>>(a.part_o, a.part_ml, p->out, out_rows, ns);
    UPR_CUDA_CHECK(cudaGetLastError());
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

upr_status upr_kv_cache_layout(const int32_t* seq_lens, int B, int H, int d, int n_layers,
                               upr_dtype dtype, upr_kv_layout* out, int64_t* row_off) {
  if (out == nullptr) return fail(UPR_ERR_INVALID_ARG, "out is NULL");
  if (B < 0 || H <= 0 || n_layers <= 0 || d <= 0 || (B > 0 && seq_lens == nullptr))
    return fail(UPR_ERR_INVALID_ARG, "bad sizes (B=%d H=%d d=%d n_layers=%d)", B, H, d, n_layers);
  if (d != 64 && d != 128) return fail(UPR_ERR_UNSUPPORTED, "head dim d=%d unsupported", d);
  if (dtype != UPR_F32 && dtype != UPR_BF16 && dtype != UPR_FP8_E4M3)
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
  out->bytes_scales = (dtype == UPR_FP8_E4M3) ? static_cast<int64_t>(n_layers) * H * 4 : 0;
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
  const bool fp8 = lay->dtype == UPR_FP8_E4M3;
  if (fp8 && ((k_pool && !k_scale) || (v_pool && !v_scale)))
    return fail(UPR_ERR_INVALID_ARG, "FP8 pack needs scale outputs");
  upr_status s = check_device();
  if (s != UPR_OK) return s;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t smem = (static_cast<size_t>(lay->B) + 1) * sizeof(int);
  if (smem > 40 * 1024) return fail(UPR_ERR_UNSUPPORTED, "B=%d too large for the pack kernel", lay->B);
  const int grid = sm_count() * 8;
  const int n_scale = lay->n_layers * lay->H;
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

upr_status upr_cross_attn_fwd(const void* q, const void* k_cache, const void* v_cache,
                              const int32_t* seq_lens, const int32_t* cand_offsets, float* out,
                              int B, int H, int d, upr_dtype dtype, void* stream) {
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
  p.total_q = 1;  // unknown on the host; only used to skip empty launches
  p.num_splits = 1;
  return run_attn(&p, /*have_workspace=*/false, static_cast<cudaStream_t>(stream));
}

int upr_cross_attn_num_splits(const upr_attn_params* p) {
  if (p == nullptr) return 1;
  return pick_splits(p);
}

size_t upr_cross_attn_workspace_bytes(const upr_attn_params* p) {
  if (p == nullptr || p->B < 0 || p->H <= 0 || p->n_layers <= 0 || p->total_q < 0 ||
      (p->d != 64 && p->d != 128))
    return 0;
  const int ns = pick_splits(p);
  size_t bytes = kCounterBytes;
  if (ns > 1) {
    const size_t rows = static_cast<size_t>(p->n_layers) * p->total_q * p->H;
    bytes += rows * ns * (static_cast<size_t>(p->d) + 2) * sizeof(float);
  }
  return bytes;
}

upr_status upr_cross_attn_fwd_ex(const upr_attn_params* p, void* stream) {
  return run_attn(p, /*have_workspace=*/true, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
