/*
 * upr_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64) of the ranking head's
 * cross-attention over a cached user history, written from the paper's definition
 * (/root/reference/PAPER.md, UniPinRec, arxiv/paper_2606_00422).  It exists only so
 * that tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs can check and time the CUDA path against something independent.  It shares no
 * code, header, table or constant generator with paper_2606_00422_b200/csrc and
 * neither side includes or links the other.
 *
 * Every function cites the passage it follows.  Symbols (SURVEY.md "symbol clash"):
 *   L_b  = history length of user b       (paper: n,  PAPER.md:138, 198)
 *   C_b  = number of candidates of user b (paper: k,  PAPER.md:138, 198)
 *   H, d = heads, head dim                (paper: H, D)
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): softmax rows sum to one;
 * single key returns its V row; identical keys return the mean of V; candidate
 * permutation and batch-composition invariance; equality with the dense
 * masked full-sequence attention of PAPER.md:138; equality with
 * torch.nn.functional.scaled_dot_product_attention in fp64 with an explicit mask;
 * split-K merge equals the unsplit result; E4M3 codec against torch.float8_e4m3fn and
 * constructed ties; layout tables against hand-written tiny cases.  No function in this
 * file is "parity unpinned".
 *
 * Build: gcc -O3 -fopenmp -ffp-contract=off -shared -fPIC upr_oracle.c -o libupr_oracle.so -lm
 * (-ffp-contract=off: the fp32 steps of the quantiser must round once per operation.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define UPRO_F32 0
#define UPRO_BF16 1
#define UPRO_FP8_E4M3 2
#define UPRO_FP8_E4M3_USER 3 /* E4M3 bytes, one scale per (layer, USER, head): SURVEY.md 8(f)3, reading Q18 */
#define UPRO_IS_FP8(dt) ((dt) == UPRO_FP8_E4M3 || (dt) == UPRO_FP8_E4M3_USER)

int upro_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * Storage formats -> fp64 (exact widenings).
 * ---------------------------------------------------------------------------------- */

/* bfloat16 bit pattern -> double: bf16 is the top 16 bits of an IEEE binary32. */
double upro_bf16_to_f64(uint16_t bits) {
  uint32_t w = ((uint32_t)bits) << 16;
  float f;
  memcpy(&f, &w, 4);
  return (double)f;
}

/* IEEE binary32 -> bfloat16 bits, round-to-nearest-even (inputs finite). */
uint16_t upro_f32_to_bf16(float f) {
  uint32_t w;
  memcpy(&w, &f, 4);
  uint32_t lsb = (w >> 16) & 1u;
  w += 0x7FFFu + lsb;
  return (uint16_t)(w >> 16);
}

/* FP8 E4M3 ("fn" variant: 1 sign, 4 exponent (bias 7), 3 mantissa bits; no infinities;
 * S.1111.111 is NaN; max finite 448 = 1.75 * 2^8; subnormals m * 2^-9, m = 1..7).
 * Format fixed by BASELINE.json config 4 / DESIGN.md reading Q6. */
double upro_e4m3_decode(uint8_t b) {
  int s = (b >> 7) & 1;
  int e = (b >> 3) & 0xF;
  int m = b & 7;
  double v;
  if (e == 0xF && m == 7) return NAN;
  if (e == 0)
    v = ldexp((double)m, -9); /* subnormal: (m/8) * 2^-6 */
  else
    v = ldexp(1.0 + (double)m / 8.0, e - 7);
  return s ? -v : v;
}

/* float -> E4M3 byte, round-to-nearest-even, saturating to +-448 (never NaN/Inf for
 * finite input).  Written as a search over the 127 non-negative finite codes so that it
 * is the definition of "nearest representable, ties to even mantissa", not a bit trick. */
uint8_t upro_e4m3_encode(float x) {
  uint8_t sign = 0;
  double a = (double)x;
  if (signbit(x)) {
    sign = 0x80;
    a = -a;
  }
  if (isnan(x)) return (uint8_t)(sign | 0x7F);
  if (a >= 448.0) return (uint8_t)(sign | 0x7E); /* satfinite */
  /* codes 0x00..0x7E are monotonically increasing in value; their decoded values are
   * tabulated once (same upro_e4m3_decode, only cached) so that packing 1e7 elements in a
   * test takes seconds, not minutes -- the nearest-code search itself is unchanged */
  static double table[0x7F];
  static int table_ready = 0;
  if (!table_ready) {
    for (int c = 0; c <= 0x7E; ++c) table[c] = upro_e4m3_decode((uint8_t)c);
    table_ready = 1;
  }
  int best = 0;
  double best_err = a; /* code 0 is value 0 */
  for (int c = 1; c <= 0x7E; ++c) {
    double v = table[c];
    double err = fabs(v - a);
    if (err < best_err) {
      best_err = err;
      best = c;
    } else if (err == best_err) {
      /* tie: choose the code with even mantissa LSB (consecutive codes differ in LSB) */
      if ((c & 1) == 0) best = c;
    }
  }
  return (uint8_t)(sign | best);
}

/* ------------------------------------------------------------------------------------
 * a0. Layout tables (integer, bit-exact contract).  DESIGN.md reading Q14:
 *   row_off[0] = 0, row_off[b+1] = row_off[b] + round_up(L_b, align); R = row_off[B];
 *   packed cache = [n_layers][H][R][d] elements followed by tail_rows rows of padding.
 * The pool it is gathered from is the paper's [L, S, H, n, D].
 * out7 = { R, elem_bytes, row_bytes, head_stride_bytes, layer_stride_bytes,
 *          bytes_cache (one of K or V, tail included), bytes_scales }
 * ---------------------------------------------------------------------------------- */
int upro_layout(const int32_t* seq_lens, int B, int H, int d, int n_layers, int dtype,
                int align, int tail_rows, int64_t* row_off, int64_t* out7) {
  if (B < 0 || H <= 0 || d <= 0 || n_layers <= 0 || align <= 0) return 1;
  int64_t acc = 0;
  row_off[0] = 0;
  for (int b = 0; b < B; ++b) {
    if (seq_lens[b] < 0) return 1;
    int64_t Lb = seq_lens[b];
    int64_t padded = ((Lb + align - 1) / align) * align;
    acc += padded;
    row_off[b + 1] = acc;
  }
  int64_t eb = (dtype == UPRO_F32) ? 4 : (dtype == UPRO_BF16) ? 2 : 1;
  out7[0] = acc;
  out7[1] = eb;
  out7[2] = eb * d;
  out7[3] = acc * eb * d;
  out7[4] = (int64_t)H * acc * eb * d;
  out7[5] = ((int64_t)n_layers * H * acc + tail_rows) * eb * d;
  out7[6] = (dtype == UPRO_FP8_E4M3) ? (int64_t)n_layers * H * 4
            : (dtype == UPRO_FP8_E4M3_USER) ? (int64_t)n_layers * B * H * 4 : 0;
  return 0;
}

/* ------------------------------------------------------------------------------------
 * a1. Pack: "each ranking consumer copies each request's past KV from its slot in the
 * mapped pool into its own decode cache".  Pool [n_layers,S,H,n_max,d]
 * bf16; user b's valid rows are [0, L_b) of slot slot_ids[b] (reading Q7).
 * Output: packed [n_layers,H,R,d] (+tail), padding rows and tail zero-filled.
 *  - dtype BF16: verbatim 16-bit copy.
 *  - dtype FP8_E4M3 (reading Q6): per (layer, head) amax over all users' valid rows;
 *    scale = amax / 448.0f (fp32 divide), amax == 0 -> scale = 1;
 *    byte = e4m3_rne_satfinite( x * (448.0f / amax) ) with the product in fp32
 *    (amax == 0 -> multiplier 1).
 * One pool (K or V) per call.
 * ---------------------------------------------------------------------------------- */
int upro_pack(const uint16_t* pool, int n_layers, int S, int H, int n_max, int d,
              const int32_t* slot_ids, const int32_t* seq_lens, int B, int dtype, int align,
              int tail_rows, void* cache, float* scales) {
  int64_t* row_off = (int64_t*)malloc(sizeof(int64_t) * (size_t)(B + 1));
  int64_t o7[7];
  if (upro_layout(seq_lens, B, H, d, n_layers, dtype, align, tail_rows, row_off, o7)) {
    free(row_off);
    return 1;
  }
  int64_t R = o7[0];
  memset(cache, 0, (size_t)o7[5]);
  for (int l = 0; l < n_layers; ++l)
    for (int h = 0; h < H; ++h) {
      float mult = 1.0f;
      if (dtype == UPRO_FP8_E4M3) {
        float amax = 0.0f;
        for (int b = 0; b < B; ++b) {
          const uint16_t* src =
              pool + ((((int64_t)l * S + slot_ids[b]) * H + h) * n_max) * (int64_t)d;
          for (int64_t i = 0; i < (int64_t)seq_lens[b] * d; ++i) {
            float v = fabsf((float)upro_bf16_to_f64(src[i]));
            if (v > amax) amax = v;
          }
        }
        if (amax > 0.0f) {
          scales[l * H + h] = amax / 448.0f;
          mult = 448.0f / amax;
        } else {
          scales[l * H + h] = 1.0f;
          mult = 1.0f;
        }
      }
      for (int b = 0; b < B; ++b) {
        if (seq_lens[b] > n_max || slot_ids[b] < 0 || slot_ids[b] >= S) {
          free(row_off);
          return 1;
        }
        const uint16_t* src =
            pool + ((((int64_t)l * S + slot_ids[b]) * H + h) * n_max) * (int64_t)d;
        int64_t dst0 = (((int64_t)l * H + h) * R + row_off[b]) * (int64_t)d;
        int64_t n = (int64_t)seq_lens[b] * d;
        if (dtype == UPRO_FP8_E4M3_USER) {
          /* the same rule as above, amax over THIS user's valid rows of the (layer, head) only:
             a cache that is written user by user (incrementally) never needs another user's rows */
          float amax = 0.0f;
          for (int64_t i = 0; i < n; ++i) {
            float v = fabsf((float)upro_bf16_to_f64(src[i]));
            if (v > amax) amax = v;
          }
          int64_t si = ((int64_t)l * B + b) * H + h;
          scales[si] = amax > 0.0f ? amax / 448.0f : 1.0f;
          mult = amax > 0.0f ? 448.0f / amax : 1.0f;
        }
        if (dtype == UPRO_BF16) {
          memcpy((uint16_t*)cache + dst0, src, (size_t)n * 2);
        } else if (UPRO_IS_FP8(dtype)) {
          uint8_t* dst = (uint8_t*)cache + dst0;
          for (int64_t i = 0; i < n; ++i) {
            float x = (float)upro_bf16_to_f64(src[i]);
            volatile float y = x * mult; /* one fp32 rounding */
            dst[i] = upro_e4m3_encode(y);
          }
        } else { /* F32 cache: exact widening of the bf16 pool */
          float* dst = (float*)cache + dst0;
          for (int64_t i = 0; i < n; ++i) dst[i] = (float)upro_bf16_to_f64(src[i]);
        }
      }
    }
  free(row_off);
  return 0;
}

/* ------------------------------------------------------------------------------------
 * a2-a7. One (layer, user, head) block of the ranking head's attention, the plain
 * definition (two-pass softmax, fp64).  PAPER.md:138: "each candidate position n+j
 * attends to all past positions 1..n but is blocked from attending to other candidates";
 * "ranking attends directly to the cached history KV ... identity-mask
 * design"; ranking is "a decode step that attends from candidates into a
 * frozen history".  Softmax scaled-dot-product (readings Q1, Q2).
 *
 *   q     [C][d]   candidate queries           K, V   [L][d]  cached history keys/values
 *   kself, vself [C][d] or NULL (the candidate's own key/value: identity block of the
 *                 mask, reading Q3)
 *   out   [C][d]
 *   wout  optional [C][L+1]: normalised softmax weights (last column = self weight, 0
 *         if no self term) -- exposed so tests can check that rows sum to one.
 * No logit at all (L == 0 and no self term) -> zeros (reading Q9).
 * ---------------------------------------------------------------------------------- */
void upro_attn_block(const double* q, const double* K, const double* V, const double* kself,
                     const double* vself, int C, int L, int d, double scale, double* out,
                     double* wout) {
  double* s = (double*)malloc(sizeof(double) * (size_t)(L + 1));
  for (int c = 0; c < C; ++c) {
    const double* qc = q + (size_t)c * d;
    int has_self = (kself != NULL);
    /* step 1: logits over the history */
    for (int j = 0; j < L; ++j) {
      double acc = 0.0;
      for (int t = 0; t < d; ++t) acc += qc[t] * K[(size_t)j * d + t];
      s[j] = scale * acc;
    }
    /* step 2: self logit */
    double s_self = 0.0;
    if (has_self) {
      double acc = 0.0;
      for (int t = 0; t < d; ++t) acc += qc[t] * kself[(size_t)c * d + t];
      s_self = scale * acc;
    }
    double* o = out + (size_t)c * d;
    for (int t = 0; t < d; ++t) o[t] = 0.0;
    if (wout)
      for (int j = 0; j <= L; ++j) wout[(size_t)c * (L + 1) + j] = 0.0;
    if (L == 0 && !has_self) continue;
    /* step 3: max, weights, normaliser */
    double m = has_self ? s_self : s[0];
    for (int j = 0; j < L; ++j)
      if (s[j] > m) m = s[j];
    double Z = 0.0;
    for (int j = 0; j < L; ++j) {
      s[j] = exp(s[j] - m);
      Z += s[j];
    }
    double w_self = 0.0;
    if (has_self) {
      w_self = exp(s_self - m);
      Z += w_self;
    }
    /* step 4: weighted sum of values */
    for (int j = 0; j < L; ++j)
      for (int t = 0; t < d; ++t) o[t] += s[j] * V[(size_t)j * d + t];
    if (has_self)
      for (int t = 0; t < d; ++t) o[t] += w_self * vself[(size_t)c * d + t];
    for (int t = 0; t < d; ++t) o[t] /= Z;
    if (wout) {
      for (int j = 0; j < L; ++j) wout[(size_t)c * (L + 1) + j] = s[j] / Z;
      wout[(size_t)c * (L + 1) + L] = w_self / Z;
    }
  }
  free(s);
}

/* ------------------------------------------------------------------------------------
 * The paper's own formulation, for the equivalence pin: dense masked softmax attention
 * over the concatenated sequence [history(n) || candidates(k)]:
 *   row i <  n     : attends j <= i (standard causal)
 *   row i = n + c  : attends all j < n; attends j = n + c iff self_flag; no other j.
 * xq, xk, xv are [(n+k)][d]; out is [(n+k)][d]; mask_out (optional, [(n+k)][(n+k)]
 * bytes) receives the materialised mask so its unmasked-pair count can be checked
 * against n(n+1)/2 + nk (+k)  (O(n^2 + nk) instead of O((n+k)^2)).
 * ---------------------------------------------------------------------------------- */
void upro_full_sequence_attention(const double* xq, const double* xk, const double* xv, int n,
                                  int k, int d, int self_flag, double scale, double* out,
                                  uint8_t* mask_out) {
  int T = n + k;
  uint8_t* mask = (uint8_t*)calloc((size_t)T * T, 1);
  for (int i = 0; i < T; ++i)
    for (int j = 0; j < T; ++j) {
      uint8_t a;
      if (i < n)
        a = (j <= i);
      else if (j < n)
        a = 1;
      else
        a = (uint8_t)(self_flag && j == i);
      mask[(size_t)i * T + j] = a;
    }
  double* s = (double*)malloc(sizeof(double) * (size_t)T);
  for (int i = 0; i < T; ++i) {
    double m = -INFINITY;
    int any = 0;
    for (int j = 0; j < T; ++j) {
      if (!mask[(size_t)i * T + j]) continue;
      double acc = 0.0;
      for (int t = 0; t < d; ++t) acc += xq[(size_t)i * d + t] * xk[(size_t)j * d + t];
      s[j] = scale * acc;
      if (s[j] > m) m = s[j];
      any = 1;
    }
    for (int t = 0; t < d; ++t) out[(size_t)i * d + t] = 0.0;
    if (!any) continue;
    double Z = 0.0;
    for (int j = 0; j < T; ++j) {
      if (!mask[(size_t)i * T + j]) continue;
      s[j] = exp(s[j] - m);
      Z += s[j];
    }
    for (int j = 0; j < T; ++j) {
      if (!mask[(size_t)i * T + j]) continue;
      for (int t = 0; t < d; ++t) out[(size_t)i * d + t] += s[j] * xv[(size_t)j * d + t];
    }
    for (int t = 0; t < d; ++t) out[(size_t)i * d + t] /= Z;
  }
  if (mask_out) memcpy(mask_out, mask, (size_t)T * T);
  free(mask);
  free(s);
}

/* ------------------------------------------------------------------------------------
 * a8. Split-K partial state and its combine (north_star "split-K variant ... and its
 * combine"; long histories).  For a key range [j0, j1) of one block:
 *   m_i = max_j s_j   (natural-log units, logits already scaled)
 *   l_i = sum_j exp(s_j - m_i)
 *   Ot_i = sum_j exp(s_j - m_i) V_j            (un-normalised)
 * An empty range has m_i = -inf, l_i = 0, Ot_i = 0.  The self term, when present, is a
 * one-key range of its own (upro_attn_partial with L = 1 on kself/vself rows).
 * Combine:  m* = max_i m_i;  l* = sum_i l_i exp(m_i - m*);
 *           out = sum_i Ot_i exp(m_i - m*) / l*;   all ranges empty -> zeros.
 * ---------------------------------------------------------------------------------- */
void upro_attn_partial(const double* q, const double* K, const double* V, int C, int j0, int j1,
                       int d, double scale, double* m_out, double* l_out, double* Ot) {
  for (int c = 0; c < C; ++c) {
    const double* qc = q + (size_t)c * d;
    double m = -INFINITY;
    for (int j = j0; j < j1; ++j) {
      double acc = 0.0;
      for (int t = 0; t < d; ++t) acc += qc[t] * K[(size_t)j * d + t];
      double sj = scale * acc;
      if (sj > m) m = sj;
    }
    double l = 0.0;
    for (int t = 0; t < d; ++t) Ot[(size_t)c * d + t] = 0.0;
    for (int j = j0; j < j1; ++j) {
      double acc = 0.0;
      for (int t = 0; t < d; ++t) acc += qc[t] * K[(size_t)j * d + t];
      double w = exp(scale * acc - m);
      l += w;
      for (int t = 0; t < d; ++t) Ot[(size_t)c * d + t] += w * V[(size_t)j * d + t];
    }
    m_out[c] = m;
    l_out[c] = l;
  }
}

/* parts laid out [n_parts][C] for m, l and [n_parts][C][d] for Ot */
void upro_combine(const double* m, const double* l, const double* Ot, int n_parts, int C, int d,
                  double* out) {
  for (int c = 0; c < C; ++c) {
    double mstar = -INFINITY;
    for (int i = 0; i < n_parts; ++i)
      if (m[(size_t)i * C + c] > mstar) mstar = m[(size_t)i * C + c];
    double* o = out + (size_t)c * d;
    for (int t = 0; t < d; ++t) o[t] = 0.0;
    if (mstar == -INFINITY) continue;
    double lstar = 0.0;
    for (int i = 0; i < n_parts; ++i) {
      double mi = m[(size_t)i * C + c];
      if (mi == -INFINITY) continue;
      double f = exp(mi - mstar);
      lstar += l[(size_t)i * C + c] * f;
      for (int t = 0; t < d; ++t) o[t] += Ot[((size_t)i * C + c) * d + t] * f;
    }
    for (int t = 0; t < d; ++t) o[t] /= lstar;
  }
}

/* ------------------------------------------------------------------------------------
 * Whole batch over the packed ragged layout: every (layer, user, head) block through
 * upro_attn_block.  Inputs are the stored values the GPU consumes, widened exactly:
 *   q, kself, vself : [n_layers][total_q][H][d], q_dtype F32 (float) or BF16 (uint16 bits)
 *   k_cache, v_cache: [n_layers][H][R][d] in kv_dtype (F32 / BF16 bits / E4M3 bytes);
 *                     FP8: value = decode(byte) * scale[layer*H + h]  (exact in fp64)
 *   out             : [n_layers][total_q][H][d] fp64
 * OpenMP over (layer, user, head) blocks -- the only parallelism; arithmetic per block is
 * upro_attn_block's.  users_lo/users_hi restrict to a user range (bench sample).
 * ---------------------------------------------------------------------------------- */
static double load_elem(const void* p, int dtype, int64_t i, double scale) {
  if (dtype == UPRO_F32) return (double)((const float*)p)[i];
  if (dtype == UPRO_BF16) return upro_bf16_to_f64(((const uint16_t*)p)[i]);
  return upro_e4m3_decode(((const uint8_t*)p)[i]) * scale;
}

int upro_cross_attn_packed(const void* q, int q_dtype, const void* k_cache, const void* v_cache,
                           int kv_dtype, const float* k_scale, const float* v_scale,
                           const void* kself, const void* vself, const int32_t* seq_lens,
                           const int32_t* cand_offsets, int B, int H, int d, int n_layers,
                           int align, double sm_scale, int users_lo, int users_hi, double* out) {
  int64_t* row_off = (int64_t*)malloc(sizeof(int64_t) * (size_t)(B + 1));
  int64_t o7[7];
  if (upro_layout(seq_lens, B, H, d, n_layers, kv_dtype, align, 0, row_off, o7)) {
    free(row_off);
    return 1;
  }
  int64_t R = o7[0];
  int64_t total_q = cand_offsets[B];
  if (users_lo < 0) users_lo = 0;
  if (users_hi > B) users_hi = B;
  int64_t n_blocks = (int64_t)n_layers * (users_hi - users_lo) * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t blk = 0; blk < n_blocks; ++blk) {
    int h = (int)(blk % H);
    int b = users_lo + (int)((blk / H) % (users_hi - users_lo));
    int l = (int)(blk / ((int64_t)H * (users_hi - users_lo)));
    int C = cand_offsets[b + 1] - cand_offsets[b];
    int L = seq_lens[b];
    if (C <= 0) continue;
    int64_t si = (kv_dtype == UPRO_FP8_E4M3_USER) ? ((int64_t)l * B + b) * H + h : (int64_t)l * H + h;
    double ks = (UPRO_IS_FP8(kv_dtype) && k_scale) ? (double)k_scale[si] : 1.0;
    double vs = (UPRO_IS_FP8(kv_dtype) && v_scale) ? (double)v_scale[si] : 1.0;
    double* qb = (double*)malloc(sizeof(double) * (size_t)C * d);
    double* ob = (double*)malloc(sizeof(double) * (size_t)C * d);
    double* Kb = (double*)malloc(sizeof(double) * (size_t)(L > 0 ? L : 1) * d);
    double* Vb = (double*)malloc(sizeof(double) * (size_t)(L > 0 ? L : 1) * d);
    double* ksb = kself ? (double*)malloc(sizeof(double) * (size_t)C * d) : NULL;
    double* vsb = kself ? (double*)malloc(sizeof(double) * (size_t)C * d) : NULL;
    for (int c = 0; c < C; ++c)
      for (int t = 0; t < d; ++t) {
        int64_t gi = ((((int64_t)l * total_q + cand_offsets[b] + c) * H) + h) * d + t;
        qb[(size_t)c * d + t] = load_elem(q, q_dtype, gi, 1.0);
        if (kself) {
          ksb[(size_t)c * d + t] = load_elem(kself, q_dtype, gi, 1.0);
          vsb[(size_t)c * d + t] = load_elem(vself, q_dtype, gi, 1.0);
        }
      }
    int64_t base = (((int64_t)l * H + h) * R + row_off[b]) * d;
    for (int64_t i = 0; i < (int64_t)L * d; ++i) {
      Kb[i] = load_elem(k_cache, kv_dtype, base + i, ks);
      Vb[i] = load_elem(v_cache, kv_dtype, base + i, vs);
    }
    upro_attn_block(qb, Kb, Vb, ksb, vsb, C, L, d, sm_scale, ob, NULL);
    for (int c = 0; c < C; ++c)
      for (int t = 0; t < d; ++t) {
        int64_t gi = ((((int64_t)l * total_q + cand_offsets[b] + c) * H) + h) * d + t;
        out[gi] = ob[(size_t)c * d + t];
      }
    free(qb);
    free(ob);
    free(Kb);
    free(Vb);
    free(ksb);
    free(vsb);
  }
  free(row_off);
  return 0;
}

/* ------------------------------------------------------------------------------------
 * Whole batch straight from the paper's pool (zero-copy addressing): the
 * history K/V of user b are rows [0, L_b) of slot slot_ids[b] of the pool
 * [n_layers][S][H_kv][n_max][d] ("[L,S,H,n,D] ... KV heads"), read in place
 * instead of through the slot copy of PAPER.md:204.  Grouped queries ("KV
 * heads", reading Q5): query head hq attends over KV head hq / (H_q / H_kv); H_q == H_kv is
 * the ungrouped case.  Plain indexing + upro_attn_block, nothing else.
 *   q, kself, vself : [n_layers][total_q][H_q][d], q_dtype F32 or BF16 bits
 *   k_pool, v_pool  : bf16 bits
 *   out             : [n_layers][total_q][H_q][d] fp64
 * Returns 1 on invalid arguments (H_q not a multiple of H_kv, slot or length out of range).
 * ---------------------------------------------------------------------------------- */
int upro_cross_attn_pool(const void* q, int q_dtype, const uint16_t* k_pool,
                         const uint16_t* v_pool, int n_layers, int S, int H_kv, int n_max, int d,
                         int H_q, const int32_t* slot_ids, const int32_t* seq_lens,
                         const int32_t* cand_offsets, int B, const void* kself, const void* vself,
                         double sm_scale, int users_lo, int users_hi, double* out) {
  if (H_kv <= 0 || H_q <= 0 || H_q % H_kv != 0) return 1;
  for (int b = 0; b < B; ++b)
    if (seq_lens[b] < 0 || seq_lens[b] > n_max || slot_ids[b] < 0 || slot_ids[b] >= S) return 1;
  int G = H_q / H_kv;
  int64_t total_q = cand_offsets[B];
  if (users_lo < 0) users_lo = 0;
  if (users_hi > B) users_hi = B;
  int64_t n_blocks = (int64_t)n_layers * (users_hi - users_lo) * H_q;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t blk = 0; blk < n_blocks; ++blk) {
    int hq = (int)(blk % H_q);
    int b = users_lo + (int)((blk / H_q) % (users_hi - users_lo));
    int l = (int)(blk / ((int64_t)H_q * (users_hi - users_lo)));
    int hk = hq / G;
    int C = cand_offsets[b + 1] - cand_offsets[b];
    int L = seq_lens[b];
    if (C <= 0) continue;
    double* qb = (double*)malloc(sizeof(double) * (size_t)C * d);
    double* ob = (double*)malloc(sizeof(double) * (size_t)C * d);
    double* Kb = (double*)malloc(sizeof(double) * (size_t)(L > 0 ? L : 1) * d);
    double* Vb = (double*)malloc(sizeof(double) * (size_t)(L > 0 ? L : 1) * d);
    double* ksb = kself ? (double*)malloc(sizeof(double) * (size_t)C * d) : NULL;
    double* vsb = kself ? (double*)malloc(sizeof(double) * (size_t)C * d) : NULL;
    for (int c = 0; c < C; ++c)
      for (int t = 0; t < d; ++t) {
        int64_t gi = ((((int64_t)l * total_q + cand_offsets[b] + c) * H_q) + hq) * d + t;
        qb[(size_t)c * d + t] = load_elem(q, q_dtype, gi, 1.0);
        if (kself) {
          ksb[(size_t)c * d + t] = load_elem(kself, q_dtype, gi, 1.0);
          vsb[(size_t)c * d + t] = load_elem(vself, q_dtype, gi, 1.0);
        }
      }
    int64_t base = ((((int64_t)l * S + slot_ids[b]) * H_kv + hk) * n_max) * (int64_t)d;
    for (int64_t i = 0; i < (int64_t)L * d; ++i) {
      Kb[i] = upro_bf16_to_f64(k_pool[base + i]);
      Vb[i] = upro_bf16_to_f64(v_pool[base + i]);
    }
    upro_attn_block(qb, Kb, Vb, ksb, vsb, C, L, d, sm_scale, ob, NULL);
    for (int c = 0; c < C; ++c)
      for (int t = 0; t < d; ++t) {
        int64_t gi = ((((int64_t)l * total_q + cand_offsets[b] + c) * H_q) + hq) * d + t;
        out[gi] = ob[(size_t)c * d + t];
      }
    free(qb);
    free(ob);
    free(Kb);
    free(Vb);
    free(ksb);
    free(vsb);
  }
  return 0;
}

/* ====================================================================================
 * The rest of the ranking decode layer and its consumer.
 * ==================================================================================== */

/* ------------------------------------------------------------------------------------
 * upro_linear -- one linear layer of the ranking pass over candidate tokens only
 * ("only the candidate tokens are processed"): y = act(x W^T + b), the plain
 * definition, fp64.  W is [N, K] row-major (one output feature per row, the nn.Linear
 * convention); act: 0 = identity, 1 = SiLU x*sigmoid(x), 2 = ReLU.  The paper names no
 * activation for its MLPs (reading Q15): SiLU is this build's default.
 *   x [M, K], w [N, K], b [N] or NULL, y [M, N]
 * ---------------------------------------------------------------------------------- */
void upro_linear(const double* x, const double* w, const double* b, int64_t M, int N, int K,
                 int act, double* y) {
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < M; ++m)
    for (int n = 0; n < N; ++n) {
      double acc = 0.0;
      for (int k = 0; k < K; ++k) acc += x[m * K + k] * w[(int64_t)n * K + k];
      if (b) acc += b[n];
      if (act == 1) acc = acc / (1.0 + exp(-acc));
      else if (act == 2) acc = acc > 0.0 ? acc : 0.0;
      y[m * N + n] = acc;
    }
}

/* ------------------------------------------------------------------------------------
 * upro_action_utility -- the ranking head's consumer (PAPER.md:146-152, Eq. 4; :321).
 * For every candidate hidden state z and action type c = 0..C-1 a dedicated two-layer MLP
 * head h_c produces a scalar logit,
 *     hid_c = act(W1_c z + b1_c)   (W1_c [Dh, D], act as in upro_linear)
 *     logit_c = <w2_c, hid_c> + b2_c
 * p_c = sigmoid(logit_c) is the action probability (the BCE of Eq. 4 trains exactly this),
 * and the candidate's utility is the weighted sum  u = sum_c w_c p_c  ("head utility
 * functions"; the weights are the per-head w_c of Eq. 4 -- reading Q16).
 *   z [M, D]; w1 [C, Dh, D]; b1 [C, Dh]; w2 [C, Dh]; b2 [C]; wc [C]
 *   probs [M, C] (may be NULL), util [M]
 * ---------------------------------------------------------------------------------- */
void upro_action_utility(const double* z, const double* w1, const double* b1, const double* w2,
                         const double* b2, const double* wc, int64_t M, int D, int C, int Dh,
                         int act, double* probs, double* util) {
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < M; ++m) {
    double u = 0.0;
    for (int c = 0; c < C; ++c) {
      double logit = b2[c];
      for (int j = 0; j < Dh; ++j) {
        double h = b1[(int64_t)c * Dh + j];
        for (int t = 0; t < D; ++t) h += w1[((int64_t)c * Dh + j) * D + t] * z[m * D + t];
        if (act == 1) h = h / (1.0 + exp(-h));
        else if (act == 2) h = h > 0.0 ? h : 0.0;
        logit += w2[(int64_t)c * Dh + j] * h;
      }
      double p = 1.0 / (1.0 + exp(-logit));
      if (probs) probs[m * C + c] = p;
      u += wc[c] * p;
    }
    util[m] = u;
  }
}

/* ------------------------------------------------------------------------------------
 * upro_topk_per_user -- "returns the top K ranked candidates": for user b
 * the min(K, C_b) candidates of [cand_offsets[b], cand_offsets[b+1]) with the largest
 * utility, in descending order of utility; equal utilities in ascending order of index
 * (the order is then unique, so the comparison with the GPU is exact).  Utilities are
 * compared as the fp32 values the GPU holds.  out_idx [B, K] global candidate indices,
 * -1 past the user's count; out_cnt [B].
 * ---------------------------------------------------------------------------------- */
void upro_topk_per_user(const float* util, const int32_t* cand_offsets, int B, int K,
                        int32_t* out_idx, int32_t* out_cnt) {
  for (int b = 0; b < B; ++b) {
    int c0 = cand_offsets[b], n = cand_offsets[b + 1] - c0;
    int kk = n < K ? n : K;
    out_cnt[b] = kk;
    char* used = (char*)calloc((size_t)(n > 0 ? n : 1), 1);
    for (int r = 0; r < K; ++r) {
      int best = -1;
      if (r < kk)
        for (int i = 0; i < n; ++i) {   /* selection by repeated maximum: first index wins ties */
          if (used[i]) continue;
          if (best < 0 || util[c0 + i] > util[c0 + best]) best = i;
        }
      if (best >= 0) used[best] = 1;
      out_idx[(int64_t)b * K + r] = best >= 0 ? c0 + best : -1;
    }
    free(used);
  }
}

/* ------------------------------------------------------------------------------------
 * upro_layernorm -- layer normalisation of one token's hidden vector (PAPER.md:206 names
 * "fused modules that combine layer normalization, linear projection, and activation"):
 *     y = (x - mean(x)) / sqrt(var(x) + eps) * gamma + beta,   var = mean((x - mean)^2)
 * the textbook definition, fp64, two passes.  x, y [M, D]; gamma, beta [D].
 * ---------------------------------------------------------------------------------- */
void upro_layernorm(const double* x, const double* gamma, const double* beta, int64_t M, int D,
                    double eps, double* y) {
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < M; ++m) {
    double mean = 0.0, var = 0.0;
    for (int t = 0; t < D; ++t) mean += x[m * D + t];
    mean /= D;
    for (int t = 0; t < D; ++t) {
      double c = x[m * D + t] - mean;
      var += c * c;
    }
    var /= D;
    double r = 1.0 / sqrt(var + eps);
    for (int t = 0; t < D; ++t) y[m * D + t] = (x[m * D + t] - mean) * r * gamma[t] + beta[t];
  }
}

/* ------------------------------------------------------------------------------------
 * upro_linear_fp8q -- the same layer when the activations ARRIVE as E4M3 bytes (the output
 * of an FP8 layer before it, quantised there with x_scale, reading Q20):
 *     y[m,n] = act( x_scale * w_scale * sum_k dec(x8[m,k]) * dec(w8[n,k]) + b[n] )
 * x8 [M,K], w8 [N,K] E4M3 bytes.  fp64 accumulation (every product of two E4M3 values and
 * their sums over K <= 2^20 terms are exact in fp64).
 * ---------------------------------------------------------------------------------- */
void upro_linear_fp8q(const uint8_t* x8, float x_scale, const uint8_t* w8, float w_scale,
                      const double* b, int64_t M, int N, int K, int act, double* y) {
  double s = (double)x_scale * (double)w_scale;
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < M; ++m)
    for (int n = 0; n < N; ++n) {
      double acc = 0.0;
      for (int k = 0; k < K; ++k)
        acc += upro_e4m3_decode(x8[m * K + k]) * upro_e4m3_decode(w8[(int64_t)n * K + k]);
      acc *= s;
      if (b) acc += b[n];
      if (act == 1) acc = acc / (1.0 + exp(-acc));
      else if (act == 2) acc = acc > 0.0 ? acc : 0.0;
      y[m * N + n] = acc;
    }
}

/* ------------------------------------------------------------------------------------
 * upro_linear_fp8 -- a linear layer with FP8 E4M3 operands and fused per-tensor scaling
 * (FP8 forward in E4M3; reading Q20):
 *     q(x)   = e4m3_rne_satfinite( x * (1.0f / x_scale) )      product rounded once in fp32
 *     y[m,n] = act( x_scale * w_scale * sum_k dec(q(x)[m,k]) * dec(w8[n,k]) + b[n] )
 * x [M,K] fp32 values (the bf16 activations widened), w8 [N,K] E4M3 bytes.  fp64 accumulation.
 * ---------------------------------------------------------------------------------- */
void upro_linear_fp8(const float* x, float x_scale, const uint8_t* w8, float w_scale,
                     const double* b, int64_t M, int N, int K, int act, double* y) {
  float mult = 1.0f / x_scale;
  double* xq = (double*)malloc(sizeof(double) * (size_t)M * K);
  double* wq = (double*)malloc(sizeof(double) * (size_t)N * K);
  for (int64_t i = 0; i < M * (int64_t)K; ++i) {
    volatile float p = x[i] * mult; /* one fp32 rounding */
    xq[i] = upro_e4m3_decode(upro_e4m3_encode(p));
  }
  for (int64_t i = 0; i < (int64_t)N * K; ++i) wq[i] = upro_e4m3_decode(w8[i]);
  double s = (double)x_scale * (double)w_scale;
#pragma omp parallel for schedule(static)
  for (int64_t m = 0; m < M; ++m)
    for (int n = 0; n < N; ++n) {
      double acc = 0.0;
      for (int k = 0; k < K; ++k) acc += xq[m * K + k] * wq[(int64_t)n * K + k];
      acc *= s;
      if (b) acc += b[n];
      if (act == 1) acc = acc / (1.0 + exp(-acc));
      else if (act == 2) acc = acc > 0.0 ? acc : 0.0;
      y[m * N + n] = acc;
    }
  free(xq);
  free(wq);
}
