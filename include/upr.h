/*
 * upr.h -- C ABI of libupr: B200 (sm_100a) ranking cross-attention over a shared user-history
 * KV cache, the serving hot path of UniPinRec (arxiv/paper_2606_00422; citations below are
 * lines of /root/reference/PAPER.md).
 *
 * What the path computes: for every user b, each of that
 * user's C_b candidate items attends -- softmax scaled-dot-product attention -- over the
 * user's L_b cached, candidate-independent history keys/values, never over other
 * candidates; optionally a candidate also attends to its own key/value (the identity block
 * of the paper's M-FALCON mask).  The history K/V live in a pool written by
 * the retrieval stage, shape [layers, slots, heads, n, D], and each ranking
 * request copies its slot into a decode cache -- here a packed ragged cache.
 *
 * Conventions (all entry points):
 *  - Plain C. No exceptions cross the boundary; every function returns a upr_status and
 *    upr_last_error() returns a thread-local message for the last failure.
 *  - The caller owns all memory. The library never allocates or frees device memory.
 *    "device" pointers must be accessible from the current CUDA device; "host" pointers
 *    are ordinary host memory.
 *  - Device work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy
 *    default stream) and the calls never synchronise: they are asynchronous and CUDA-graph
 *    capturable.  No host read of any device table happens.
 *  - Only NVIDIA B200 / sm_100a is supported. There is no CPU fallback and no alternative
 *    backend: unsupported arguments return UPR_ERR_UNSUPPORTED, never a slow path.
 *  - Head dim d must be 64 or 128.
 *
 * Packed cache layout ("decode cache"; upr_kv_cache_layout describes it):
 *    element (layer l, head h, user b, key j, t) of K (or V) is at element index
 *        ((l*H + h) * R + row_off[b] + j) * d + t
 *    row_off[0] = 0, row_off[b+1] = row_off[b] + round_up(L_b, UPR_ROW_ALIGN), R = row_off[B].
 *    The rows [L_b, round_up(L_b,16)) of each user must hold finite values (upr_kv_pack
 *    writes zeros).  After the last (layer, head) block the buffer extends by
 *    UPR_TAIL_ROWS rows (any content; they are read by the last tile's TMA box, never
 *    used).  A cache buffer must therefore be at least layout.bytes_cache bytes and
 *    128-byte aligned (torch allocations are).
 */
#ifndef UPR_H_
#define UPR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  UPR_OK = 0,
  UPR_ERR_INVALID_ARG = 1, /* NULL where not allowed, negative size, bad enum */
  UPR_ERR_UNSUPPORTED = 2, /* d not in {64,128}, dtype combination not implemented */
  UPR_ERR_WORKSPACE = 3,   /* workspace missing or too small */
  UPR_ERR_CUDA = 4         /* a CUDA runtime/driver call failed (message in upr_last_error) */
} upr_status;

/* UPR_FP8_E4M3: E4M3 bytes with one fp32 scale per (layer, head); UPR_FP8_E4M3_USER: the same bytes format with
 * one scale per (layer, USER, head) -- amax over that user's valid rows only, for caches written user by user
 * (SURVEY.md 8(f)3).  Scale tables: fp32 [n_layers, H] resp. [n_layers, B, H]. */
typedef enum { UPR_F32 = 0, UPR_BF16 = 1, UPR_FP8_E4M3 = 2, UPR_FP8_E4M3_USER = 3 } upr_dtype;
typedef enum { UPR_KV_PACKED = 0, UPR_KV_POOL = 1 } upr_kv_source;
typedef enum { UPR_KERNEL_AUTO = 0, UPR_KERNEL_SINGLE = 1, UPR_KERNEL_PAIR = 2 } upr_kernel_choice;

#define UPR_ROW_ALIGN 16  /* rows; every user's block starts on a multiple of this */
#define UPR_TAIL_ROWS 128 /* rows of slack after the last block (one TMA box) */

/* Integer description of a packed cache. All sizes in bytes unless named *_rows / R. */
typedef struct upr_kv_layout {
  int32_t B, H, d, n_layers;
  int32_t dtype;      /* upr_dtype of the cache elements */
  int32_t row_align;  /* = UPR_ROW_ALIGN */
  int32_t tail_rows;  /* = UPR_TAIL_ROWS */
  int32_t elem_bytes; /* 4, 2 or 1 */
  int64_t R;          /* rows per (layer, head) block = sum_b round_up(L_b, row_align) */
  int64_t row_bytes;
  int64_t head_stride_bytes;
  int64_t layer_stride_bytes;
  int64_t bytes_cache;  /* bytes of ONE cache (K or V), tail rows included */
  int64_t bytes_scales; /* bytes of ONE scale table: n_layers*H*4 (FP8), n_layers*B*H*4 (FP8 per user), else 0 */
} upr_kv_layout;

/*
 * a0 -- layout / offsets (integer only, host only, deterministic; the CPU oracle mirrors it
 * bit for bit).  PAPER.md:202-204 fixes the pool; the ragged packed form is this library's.
 *   seq_lens  host  [B] history lengths L_b >= 0
 *   out       host  receives the layout
 *   row_off   host  [B+1] receives the row offsets, or NULL
 * Errors: INVALID_ARG for NULL out / negative sizes or lengths; UNSUPPORTED for d or dtype.
 * B == 0 is valid (R = 0).
 */
upr_status upr_kv_cache_layout(const int32_t* seq_lens, int B, int H, int d, int n_layers,
                               upr_dtype dtype, upr_kv_layout* out, int64_t* row_off);

/*
 * a1 -- pack: the slot -> decode-cache copy of PAPER.md:204 ("each ranking consumer copies
 * each request's past KV from its slot in the mapped pool into its own decode cache").
 *   k_pool, v_pool  device  bf16 [n_layers, S, H, n_max, d]  (PAPER.md:202 [L,S,H,n,D]);
 *                           user b's valid rows are [0, L_b) of slot slot_ids[b]
 *   slot_ids        device  int32 [B], each in [0, S)
 *   seq_lens        device  int32 [B], each in [0, n_max]
 *   layout          host    from upr_kv_cache_layout for the same lengths
 *   k_cache,v_cache device  layout->bytes_cache bytes each; fully written (valid rows,
 *                           zeroed alignment padding and tail)
 *   k_scale,v_scale device  fp32 [n_layers*H]; written when layout->dtype is FP8, else
 *                           ignored (may be NULL)
 * dtype BF16: bit-exact 16-bit copy.  dtype F32: exact widening.  dtype FP8_E4M3 (format
 * "fn": max finite 448, no infinities): per (layer, head) amax over all users' valid
 * rows; scale = amax / 448.0f (fp32 divide; amax == 0 -> 1.0f); stored byte =
 * cvt.rn.satfinite.e4m3( x * (448.0f / amax) ) with the product rounded once in fp32.
 * Either pool/cache pair may be NULL to pack only the other.
 */
upr_status upr_kv_pack(const void* k_pool, const void* v_pool, int S, int n_max,
                       const int32_t* slot_ids, const int32_t* seq_lens,
                       const upr_kv_layout* layout, void* k_cache, void* v_cache, float* k_scale,
                       float* v_scale, void* stream);

/*
 * a2-a7 -- the named entry point: one layer, softmax scale 1/sqrt(d), no self term,
 * no split-K.  For every user b and candidate c in [cand_offsets[b], cand_offsets[b+1]):
 *     out[c,h,:] = softmax_j( q[c,h,:] . K[b,h,j,:] / sqrt(d) ) @ V[b,h,:,:],  j < L_b
 * (PAPER.md:138, 198, 255).  A candidate with no key at all gets zeros.
 *   q            device  [total_q, H, d] row-major; bf16, or fp32 when dtype == UPR_F32
 *   k_cache,v_cache device packed cache of `dtype` for ONE layer (layout above, n_layers=1);
 *                   FP8 caches are read with unit scales here (use _ex for scales)
 *   seq_lens     device  int32 [B]
 *   cand_offsets device  int32 [B+1], non-decreasing, [0] = 0, [B] = total_q
 *   out          device  fp32 [total_q, H, d]
 * B == 0 returns UPR_OK without a launch.
 * Not a slow path: the call reads total_q = cand_offsets[B] back from the device (4 bytes, ONE
 * synchronisation of `stream`), takes a workspace the library owns (one per device and stream, grown on
 * demand, freed when the library is unloaded) and then runs exactly what upr_cross_attn_fwd_ex runs: the
 * device-built longest-first work list, the dynamic scheduler, TMA q / out tiles, the CTA-pair kernel where it
 * applies.  While `stream` is being captured into a CUDA graph the read-back is impossible: the call then
 * launches the 1-CTA kernel on its static schedule (no workspace, no host read) -- same results, slower on
 * ragged batches; use upr_cross_attn_fwd_ex in graphs.  The caches' sizes are not arguments here, so they
 * cannot be checked: upr_cross_attn_fwd_ex with kv_bytes does.
 */
upr_status upr_cross_attn_fwd(const void* q, const void* k_cache, const void* v_cache,
                              const int32_t* seq_lens, const int32_t* cand_offsets, float* out,
                              int B, int H, int d, upr_dtype dtype, void* stream);

/* Extended call: layers, self term, FP8 scales, split-K. Zero-initialise, then fill. */
typedef struct upr_attn_params {
  const void* q;               /* device [n_layers, total_q, H, d], q_dtype */
  const void* k_cache;         /* device packed cache, kv_dtype */
  const void* v_cache;
  const int32_t* seq_lens;     /* device [B] */
  const int32_t* cand_offsets; /* device [B+1] */
  float* out;                  /* device fp32 [n_layers, total_q, H, d] */
  const void* k_self;          /* device, same shape/dtype as q, or NULL: the candidate's own */
  const void* v_self;          /*   key/value joins its softmax (PAPER.md:198 identity mask) */
  const float* k_scale;        /* device fp32 [n_layers*H] ([n_layers*B*H] for UPR_FP8_E4M3_USER) or NULL (=1) */
  const float* v_scale;
  int32_t B, H, d, n_layers;
  int32_t kv_dtype;            /* upr_dtype of the caches */
  int32_t q_dtype;             /* UPR_BF16 or UPR_F32 (q, k_self, v_self) */
  int64_t total_q;             /* host copy of cand_offsets[B] */
  float sm_scale;              /* softmax scale; 0 -> 1/sqrt(d) */
  int32_t num_splits;          /* split-K factor along the history; 0 -> heuristic, 1 -> off */
  int32_t max_seq_len;         /* hint for the heuristic (0 = unknown) */
  void* workspace;             /* device, >= upr_cross_attn_workspace_bytes(), 256-B aligned; it holds the
                                  scheduler state of ONE call: two calls in flight at the same time (on
                                  different streams) must not share a workspace.  Diagnostic: after a call,
                                  bytes [64, 80) hold two uint64 written by CTA 0 of the attention kernel --
                                  the SM cycles (clock64) and the nanoseconds (%globaltimer) it ran; their
                                  ratio is the clock the SMs really ran at under the kernel */
  size_t workspace_bytes;
  /* --- fields below may be left zero: packed cache, H_kv = H, no size check ----------------- */
  int32_t kv_source;           /* UPR_KV_PACKED (0): k_cache/v_cache are packed decode caches;
                                  UPR_KV_POOL (1): k_cache/v_cache are the POOLS themselves, bf16
                                  [n_layers, pool_slots, H_kv, pool_n_max, d], read in place --
                                  no slot copy (the copy PAPER.md:204 / 278 pays for); kv_dtype must be BF16 */
  int32_t pool_slots;          /* S      (UPR_KV_POOL only) */
  int32_t pool_n_max;          /* n      (UPR_KV_POOL only); seq_lens[b] <= n */
  int32_t H_kv;                /* KV heads ("KV heads"); 0 -> H.  H % H_kv == 0: query head hq
                                  attends KV head hq / (H / H_kv) (grouped queries folded into M) */
  const int32_t* slot_ids;     /* device int32 [B], each in [0, pool_slots) (UPR_KV_POOL only) */
  int64_t kv_bytes;            /* size in bytes of EACH of k_cache / v_cache as allocated by the caller, or 0
                                  = unchecked.  When set, a buffer shorter than the layout needs (pool:
                                  n_layers*S*H_kv*n*d*2; packed cache with kv_rows set: layout.bytes_cache) is
                                  refused with UPR_ERR_INVALID_ARG, and the bf16 K/V tensor maps are clipped
                                  to it, so no TMA read ever leaves the allocation (rows beyond it read 0). */
  int64_t kv_rows;             /* packed cache: layout.R of the cache (host copy), or 0 = unknown */
  int32_t causal;              /* 1: candidate c of user b (local index cl in [0, C_b)) sees only the keys
                                  j <= cl + (L_b - C_b) -- with C_b = L_b and q = the history tokens' queries this is the
                                  causal O(n^2) self-attention of the history prefill over K/V that
                                  already sit in the pool / cache layout.  CTA-pair kernel only (bf16, d = 128), no
                                  split-K; a candidate that sees no key gets zeros (or its self term). */
  int32_t kernel;              /* UPR_KERNEL_AUTO (0): the library picks.  UPR_KERNEL_SINGLE (1) / UPR_KERNEL_PAIR
                                  (2) force the 1-CTA kernel / the CTA-pair kernel (bf16 q and K/V, d = 128,
                                  H / H_kv in {1,2,4,8}); a forced kernel that cannot run the arguments
                                  returns UPR_ERR_UNSUPPORTED.  For tests and tuning. */
} upr_attn_params;

/* Bytes of workspace upr_cross_attn_fwd_ex needs for these params (dynamic-scheduler
 * counter + split-K partial states (m, l, O~), a8). Returns 0 on invalid params. */
size_t upr_cross_attn_workspace_bytes(const upr_attn_params* p);

/* Number of history splits the heuristic picks for these params (>= 1). */
int upr_cross_attn_num_splits(const upr_attn_params* p);

/*
 * a2-a8 -- extended forward. As upr_cross_attn_fwd, per layer, plus:
 *  - self term (k_self/v_self non-NULL): logit scale*<q_c, k_self_c> joins candidate c's
 *    softmax and v_self_c its weighted sum; with L_b == 0 the output is v_self_c.
 *  - FP8: K = e4m3(byte) * k_scale[l*H+h], V likewise; dequantised in registers (exactly: one
 *    cvt to fp16 per two bytes), MMA in fp16 -- q is converted to fp16 on its way into shared
 *    memory (exact for 2^-14 <= |q| < 65504, saturating above, rounded below), the softmax
 *    weights are packed as fp16.  The cache must hold finite codes (upr_kv_pack's satfinite
 *    conversion guarantees it): the NaN code S.1111.111 is not special-cased and stays a NaN.
 *  - split-K: the history is cut into num_splits ranges of whole 128-key tiles, each CTA
 *    writes its partial (m, l, O~) to the workspace and a combine kernel merges them.
 * Errors: WORKSPACE if workspace is NULL/too small; others as above.
 */
upr_status upr_cross_attn_fwd_ex(const upr_attn_params* p, void* stream);

/*
 * The same call for callers that must not allocate (CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): identical to upr_cross_attn_fwd_ex -- same params, same kernels, same results -- except that
 * p->workspace / p->workspace_bytes are IGNORED and the scratch (scheduler counter, work-list tables, split-K
 * partials) is a static device array inside the library, UPR_NOALLOC_SCRATCH_BYTES long.  The call performs no
 * cudaMalloc / cudaFree and calls no allocating library routine; the first call on a device looks the array's
 * address up (cudaGetSymbolAddress) and keeps it.
 *   - Limit: a call whose upr_cross_attn_workspace_bytes(p) exceeds UPR_NOALLOC_SCRATCH_BYTES is refused with
 *     UPR_ERR_WORKSPACE and a message that states both numbers (without split-K the need is 256 + ~12 (B + 1)
 *     bytes; split-K adds n_layers * total_q * H * num_splits * (d + 2) * 4).
 *   - Cost: every GPU on which the library is loaded holds the array until the process exits.
 *   - ALL calls on a device share the one array: two calls that overlap on the GPU (different streams, or two
 *     host threads) race on the scheduler state and corrupt each other's results.  Order them on one stream or
 *     with events.  The array keeps the last call's contents; each call rewrites what it reads before reading it.
 */
#define UPR_NOALLOC_SCRATCH_BYTES (8u << 20)
size_t upr_cross_attn_noalloc_scratch_bytes(void);
upr_status upr_cross_attn_fwd_noalloc(const upr_attn_params* p, void* stream);

/* ====================================================================================
 * Around the attention: the rest of one ranking decode layer and the consumer
 * of the ranking pass (8(f)4).  Candidate tokens only; synthetic weights.
 * ==================================================================================== */

typedef enum { UPR_ACT_NONE = 0, UPR_ACT_SILU = 1, UPR_ACT_RELU = 2 } upr_activation;

/*
 * y = act(x W^T + bias): out-projection, MLP and projection layers of the candidate-only pass
 * (PAPER.md:192), the stacked first layers of the per-action heads.  tcgen05 GEMM,
 * bf16 operands, fp32 accumulation.
 *   x     device  [M, K] row-major, x_dtype UPR_BF16 or UPR_F32 (fp32 rows -- e.g. the attention output --
 *                 are rounded to bf16 inside the kernel on their way into the MMA, no cast pass)
 *   w     device  bf16 [N, K] row-major (one output feature per row)
 *   bias  device  fp32 [N] or NULL
 *   y     device  [M, N] row-major, y_dtype UPR_BF16 or UPR_F32
 * K % 64 == 0 and N % 8 == 0 (else UPR_ERR_UNSUPPORTED); M >= 0 (0: no launch); x, w 16-byte aligned.
 */
upr_status upr_linear_fwd(const void* x, upr_dtype x_dtype, const void* w, const float* bias, void* y,
                          upr_dtype y_dtype, int64_t M, int N, int K, upr_activation act, void* stream);
/* The same with the residual stream added after the activation: y = act(x W^T + bias) + residual, residual device
 * bf16 [M, N] (may alias y).  The out-projection and the MLP's down-projection of a decode layer. */
upr_status upr_linear_residual_fwd(const void* x, upr_dtype x_dtype, const void* w, const float* bias,
                                   const void* residual, void* y, upr_dtype y_dtype, int64_t M, int N, int K,
                                   upr_activation act, void* stream);

/*
 * FP8 linear layer with fused scaling ("mixed-precision FP8 ... E4M3 during the forward pass"; the
 * paper's are Transformer Engine modules): y = act((q(x) q(W)^T) * x_scale * w_scale + bias) [+ residual], where
 *     q(x) = cvt.rn.satfinite.e4m3(x * (1.0f / x_scale))   -- quantised INSIDE the kernel, per-tensor scale
 *     w_e4m3 = the weights already quantised to E4M3 bytes [N, K] with the per-tensor scale w_scale
 * tcgen05.mma kind::f8f6f4 on CTA pairs, fp32 accumulation.  x device bf16 [M, K]; K % 128 == 0, N % 8 == 0.
 */
upr_status upr_linear_fp8_fwd(const void* x, float x_scale, const void* w_e4m3, float w_scale, const float* bias,
                              const void* residual, void* y, upr_dtype y_dtype, int64_t M, int N, int K,
                              upr_activation act, void* stream);
/*
 * The same layer inside an FP8 CHAIN (MLP up -> down): the activations may arrive as E4M3 bytes and / or leave as
 * E4M3 bytes, so that between two FP8 layers the tensor crosses HBM once, at one byte per element, and the second
 * layer's operands both come straight through TMA (no in-kernel quantisation):
 *   x_dtype UPR_BF16      x device bf16 [M, K], quantised in the kernel with x_scale (as upr_linear_fp8_fwd)
 *           UPR_FP8_E4M3  x device E4M3 bytes [M, K], real value = dec(byte) * x_scale
 *   y_dtype UPR_BF16 / UPR_F32  as above (y_scale ignored)
 *           UPR_FP8_E4M3  y device E4M3 bytes [M, N]:
 *                         byte = cvt.rn.satfinite.e4m3( fp32(act(...) [+ residual]) * (1.0f / y_scale) )
 * K % 128 == 0, N % 8 == 0; scales > 0 (else UPR_ERR_INVALID_ARG).
 */
upr_status upr_linear_fp8_ex_fwd(const void* x, upr_dtype x_dtype, float x_scale, const void* w_e4m3, float w_scale,
                                 const float* bias, const void* residual, void* y, upr_dtype y_dtype, float y_scale,
                                 int64_t M, int N, int K, upr_activation act, void* stream);

/* Layer normalisation of candidate tokens: y = (x - mean) / sqrt(var + eps) * gamma + beta over the
 * hidden dimension; x, y device bf16 [M, D]; gamma, beta device fp32 [D]; D % 8 == 0, D <= 4096. */
upr_status upr_layernorm_fwd(const void* x, const float* gamma, const float* beta, void* y, int64_t M, int D,
                             float eps, void* stream);
/* The same with the output quantised for an FP8 layer: y_e4m3 device E4M3 bytes [M, D],
 * byte = cvt.rn.satfinite.e4m3( fp32(layer-norm value) * (1.0f / y_scale) ), y_scale > 0. */
upr_status upr_layernorm_fp8_fwd(const void* x, const float* gamma, const float* beta, void* y_e4m3, float y_scale,
                                 int64_t M, int D, float eps, void* stream);

/*
 * Prefill into the layout: the K (or V) projection of M history tokens written straight into
 * the pool [n_layers, S, H, n, d] -- no intermediate [M, H*d] tensor and no scatter pass:
 *     pool[layer, tok_slot[m], h, tok_pos[m], :] = (x[m] W^T + bias)[h*d : (h+1)*d]        (bf16)
 * Same GEMM kernel as upr_linear_fwd (N = H * d), the epilogue addresses the pool.
 *   x device [M, K] bf16 or fp32; w device bf16 [H*d, K]; bias device fp32 [H*d] or NULL
 *   pool device bf16; tok_slot, tok_pos device int32 [M] (slot in [0, S), position in [0, n))
 * The attention can then read the slot in place (kv_source = UPR_KV_POOL; causal = 1 for the prefill itself).
 */
upr_status upr_kv_project_into_pool(const void* x, upr_dtype x_dtype, const void* w, const float* bias, void* pool,
                                    const int32_t* tok_slot, const int32_t* tok_pos, int64_t M, int K, int layer,
                                    int n_layers, int S, int H, int n, int d, void* stream);

/*
 * Per-action heads, second half: hid = act(W1_c z + b1_c) for the C heads side by
 * side comes from upr_linear_fwd (N = C * Dh); this call finishes them:
 *     logit_c = <w2_c, hid_c> + b2_c,  p_c = sigmoid(logit_c),  util = sum_c wc_c * p_c
 * ("head utility functions"; wc = the per-head weights of Eq. 4).
 *   hid   device bf16 [M, C * Dh]; w2 device fp32 [C, Dh]; b2, wc device fp32 [C]
 *   probs device fp32 [M, C] or NULL; util device fp32 [M]
 * Dh % 8 == 0.
 */
upr_status upr_action_utility(const void* hid, const float* w2, const float* b2, const float* wc, int64_t M,
                              int C, int Dh, float* probs, float* util, void* stream);

/*
 * "returns the top K ranked candidates": for every user b the min(K, C_b) candidates of
 * [cand_offsets[b], cand_offsets[b+1]) with the largest utility, descending; equal utilities in
 * ascending order of candidate index (the result is unique).
 *   util device fp32 [total_q]; cand_offsets device int32 [B+1]
 *   max_cands  host upper bound on any user's candidate count (<= 16384, else UPR_ERR_UNSUPPORTED)
 *   out_idx device int32 [B, K]: global candidate indices, -1 past the user's count; out_cnt device int32 [B]
 */
upr_status upr_topk_per_user(const float* util, const int32_t* cand_offsets, int B, int K, int max_cands,
                             int32_t* out_idx, int32_t* out_cnt, void* stream);

/* ====================================================================================
 * The KV pool across processes: the retrieval replica allocates the
 * pool [L, S, H, n, D], exports a CUDA IPC handle "to a per-instance file", the ranking process opens it
 * and reads the same physical allocation in place (with UPR_KV_POOL: no copy at all); slots are reused
 * round-robin.
 * ==================================================================================== */

#define UPR_IPC_HANDLE_BYTES 80
typedef struct upr_ipc_handle { unsigned char bytes[UPR_IPC_HANDLE_BYTES]; } upr_ipc_handle;

/* Export a handle for device memory allocated in THIS process (cudaMalloc-class).  pool_dev may point
 * anywhere inside its allocation (a framework's caching allocator sub-allocates): the handle carries the
 * CUDA IPC handle of the allocation and the pointer's offset in it.  The handle is plain bytes: write it
 * to a file, a pipe, shared memory. */
upr_status upr_pool_export(const void* pool_dev, upr_ipc_handle* out);
/* Map the exporter's allocation into this (other) process; *pool_dev (the exporter's pointer, translated)
 * is valid until upr_pool_close(*pool_dev).  One open mapping per allocation and process (a CUDA rule). */
upr_status upr_pool_open(const upr_ipc_handle* handle, void** pool_dev);
upr_status upr_pool_close(void* pool_dev);

/* Round-robin slot assignment ("slots are reused round-robin"): host-only, no device work.
 * state: {S, next}; upr_slot_ring_acquire writes n consecutive slot ids (mod S) and advances. */
typedef struct upr_slot_ring { int32_t S; int32_t next; } upr_slot_ring;
upr_status upr_slot_ring_init(upr_slot_ring* ring, int32_t S);
upr_status upr_slot_ring_acquire(upr_slot_ring* ring, int32_t n, int32_t* slot_ids_host);

/* Kernel launches the last successful call on this thread enqueued (for accounting). */
int upr_last_launch_count(void);

/* Name of the attention kernel the last successful forward call on this thread launched:
 * "upr_attn_pair_kernel" (CTA pairs, tcgen05 cta_group::2) or "upr_attn_fwd_kernel" (one CTA per SM). */
const char* upr_last_attn_kernel(void);

/* Thread-local description of the last error on this thread ("" if none). */
const char* upr_last_error(void);

/* Library version string, e.g. "upr 0.1 sm_100a". */
const char* upr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* UPR_H_ */
