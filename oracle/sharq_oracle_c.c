/* SharQ CPU oracle in plain C -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A second, independent restatement of the SharQ per-linear-layer hot path (arxiv/paper_2606_26587; "P:n" = line n of
 * /root/reference/PAPER.md), written from the paper and DESIGN.md's readings R1-R8, NOT from oracle/sharq_oracle.py and
 * not from the CUDA sources: it shares no code with either.  It exists for two reasons:
 *   1. a cross-pin: tests/test_oracle_c.py requires this file and the numpy oracle to agree byte for byte on every
 *      prepared output (two independent implementations of one specification), and to 1e-12 on the fp64 linear;
 *   2. the CPU baseline BASELINE.md section 3 asks for: the oracle compiled with -O2 (no fast-math, no FMA contraction),
 *      rows parallelised over the host cores with OpenMP.  Never tuned beyond that.
 * Scope: NVFP4 and MXFP4, pairwise 4:8 mask, norm none / RMS / Layer, dynamic or static tensor scale, weights, Eq. 9 in
 * fp64, the two operators folded in front of the preparation (residual add, SiLU(gate) * up: R18), and HiF4 (Algorithm 1,
 * 2:4 mask, R9-R12) at the end of the file.  (The element-wise 2:4 mask on E2M1 formats and the Table 5 path combinations
 * live in the numpy oracle only.)
 *
 * Numerics contract (R1-R8): every float operation below is ONE IEEE-754 binary32 operation, round to nearest
 * even; build with -O2 -ffp-contract=off -fno-fast-math (oracle/build_c.py).  bf16 values travel as uint16 bit patterns.
 * Only tests/, __graft_entry__ (build / smoke) and bench.py's cpu_baseline / --impl reference legs may load this library.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { FMT_NVFP4 = 0, FMT_MXFP4 = 1 };
enum { NORM_NONE = 0, NORM_RMS = 1, NORM_LAYER = 2 };

/* ---- bit-level helpers ------------------------------------------------------------------------------------------ */
static inline float bits_f32(uint32_t u) { float f; memcpy(&f, &u, 4); return f; }
static inline uint32_t f32_bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }
static inline float bf16_to_f32(uint16_t h) { return bits_f32((uint32_t)h << 16); }
/* fp32 -> bf16, round to nearest, ties to even (finite inputs) */
static inline uint16_t f32_to_bf16(float f) {
  uint32_t u = f32_bits(f);
  uint32_t lsb = (u >> 16) & 1u;
  return (uint16_t)((u + 0x7FFFu + lsb) >> 16);
}

/* E2M1: magnitudes {0, .5, 1, 1.5, 2, 3, 4, 6}; nearest, ties to the even code, saturating; the sign bit of the
 * input survives even when the magnitude rounds to zero */
static inline uint8_t e2m1_encode(float v) {
  static const float grid[8] = {0.0f, 0.5f, 1.0f, 1.5f, 2.0f, 3.0f, 4.0f, 6.0f};
  float a = fabsf(v);
  int code = 7;
  if (a < 6.0f) {
    code = 0;
    while (code < 7 && a >= grid[code + 1]) ++code;          /* grid[code] <= a < grid[code + 1] */
    float lo = a - grid[code], hi = grid[code + 1] - a;       /* both exact: small dyadic numbers */
    if (hi < lo || (hi == lo && (code & 1))) ++code;          /* nearer neighbour; a tie goes to the even code */
  }
  return (uint8_t)(code | ((f32_bits(v) >> 31) << 3));
}
static inline float e2m1_decode(uint8_t c) {
  static const float grid[8] = {0.0f, 0.5f, 1.0f, 1.5f, 2.0f, 3.0f, 4.0f, 6.0f};
  float m = grid[c & 7];
  return (c & 8) ? -m : m;
}

/* E4M3: bias 7, 3 mantissa bits, subnormals down to 2^-9, largest finite 448; x >= 0; RNE, saturating */
static inline float e4m3_decode(uint8_t c) {
  int e = (c >> 3) & 15, m = c & 7;
  return e == 0 ? ldexpf((float)m, -9) : ldexpf((float)(8 + m), e - 10);
}
static inline uint8_t e4m3_encode(float x) {
  if (!(x > 0.0f)) return 0;
  if (x >= 448.0f) return 0x7E;
  /* walk the 127 finite codes: the grid is monotone in the code, so bisect for the last code whose value is <= x */
  int lo = 0, hi = 0x7E;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (e4m3_decode((uint8_t)mid) <= x) lo = mid; else hi = mid - 1;
  }
  if (lo == 0x7E) return 0x7E;
  double below = (double)e4m3_decode((uint8_t)lo), above = (double)e4m3_decode((uint8_t)(lo + 1));
  double dl = (double)x - below, dh = above - (double)x;      /* exact in double */
  if (dh < dl || (dh == dl && (lo & 1))) ++lo;                /* ties to the even code (even mantissa) */
  return (uint8_t)lo;
}

/* E8M0: smallest power of two >= x (x >= 0), exponent clamped to [-127, 127]; x == 0 -> 2^-127 (R8) */
static inline uint8_t e8m0_encode_up(float x) {
  if (!(x > 0.0f)) return 0;
  int e;
  float m = frexpf(x, &e);                                    /* x = m 2^e, m in [0.5, 1) */
  int up = (m == 0.5f) ? e - 1 : e;
  if (up < -127) up = -127;
  if (up > 127) up = 127;
  return (uint8_t)(up + 127);
}
static inline float e8m0_decode(uint8_t c) { return ldexpf(1.0f, (int)c - 127); }

static const uint32_t kC6bits = 0x3E2AAAABu;                  /* RN(1/6), R6 */

/* block scale (Eq. 3; R6, R8): code, effective scale and its reciprocal for a group maximum a */
static inline void block_scale(float a, int fmt, float ts, float inv_ts, uint8_t* code, float* s_eff, float* inv) {
  float q = a * bits_f32(kC6bits);
  if (fmt == FMT_NVFP4) {
    float sf = q * inv_ts;
    *code = e4m3_encode(sf);
    *s_eff = e4m3_decode(*code) * ts;
  } else {
    *code = e8m0_encode_up(q);
    *s_eff = e8m0_decode(*code);
  }
  *inv = (*s_eff == 0.0f) ? 0.0f : 1.0f / *s_eff;
}

/* ---- O1 normalisation (R1, R3) --------------------------------------------------------------- */
/* canonical fp32 sum of t[0..K) (or of RN(t*t)), in R1's order, defined on the column index k */
static float canonical_sum(const float* t, int64_t K, int squares) {
  float P[32];
  for (int l = 0; l < 32; ++l) P[l] = 0.0f;
  int64_t blocks = (K + 1023) / 1024;
  for (int64_t b = 0; b < blocks; ++b)
    for (int j = 0; j < 4; ++j)
      for (int l = 0; l < 32; ++l) {
        float leaf = 0.0f;
        for (int i = 0; i < 8; ++i) {
          int64_t k = b * 1024 + l * 32 + j * 8 + i;
          float v = k < K ? t[k] : 0.0f;                     /* columns beyond K do not exist: +0 */
          if (squares) v = v * v;
          leaf = leaf + v;
        }
        P[l] = P[l] + leaf;
      }
  for (int delta = 16; delta >= 1; delta >>= 1) {
    float Q[32];
    for (int l = 0; l < 32; ++l) Q[l] = P[l] + P[l ^ delta];
    memcpy(P, Q, sizeof P);
  }
  return P[0];
}

/* X (bf16 bits) = norm(x) for one row; c is scratch of K floats */
static void normalize_row(const uint16_t* x, int64_t K, int norm, const uint16_t* gamma, const uint16_t* beta, float eps,
                          uint16_t* X, float* c) {
  if (norm == NORM_NONE) { memcpy(X, x, (size_t)K * 2); return; }
  for (int64_t k = 0; k < K; ++k) c[k] = bf16_to_f32(x[k]);
  float Kf = (float)K;
  if (norm == NORM_LAYER) {
    float mu = canonical_sum(c, K, 0) / Kf;
    for (int64_t k = 0; k < K; ++k) c[k] = c[k] - mu;
  }
  float S = canonical_sum(c, K, 1);
  float ms = S / Kf;
  float v = ms + eps;
  float rstd = 1.0f / sqrtf(v);
  for (int64_t k = 0; k < K; ++k) {
    uint16_t h = f32_to_bf16(c[k] * rstd);                                        /* first rounding: h = bf16(x rstd) */
    uint16_t g = f32_to_bf16(bf16_to_f32(h) * bf16_to_f32(gamma[k]));             /* second: X = bf16(h gamma) */
    if (norm == NORM_LAYER && beta) g = f32_to_bf16(bf16_to_f32(g) + bf16_to_f32(beta[k]));
    X[k] = g;
  }
}

/* ---- O3 pairwise 4:8 mask (R2, R4) ---------------------------------------------------------------------- */
/* one chunk of 8 bf16 values -> the two kept pair indices i0 < i1 */
static void top2_pairs(const uint16_t* X8, int* i0, int* i1) {
  int score[4];
  for (int p = 0; p < 4; ++p) {
    int a = X8[2 * p] & 0x7FFF, b = X8[2 * p + 1] & 0x7FFF;
    score[p] = a > b ? a : b;
  }
  /* best, then second best; a later pair wins only when strictly larger, so ties go to the lower index */
  int first = 0;
  for (int p = 1; p < 4; ++p) if (score[p] > score[first]) first = p;
  int second = -1;
  for (int p = 0; p < 4; ++p) {
    if (p == first) continue;
    if (second < 0 || score[p] > score[second]) second = p;
  }
  *i0 = first < second ? first : second;
  *i1 = first < second ? second : first;
}

/* ---- sharq_prepare, one row (Fig. 2) ----------------------------------------------------------- */
static void prepare_row(const uint16_t* x, int64_t K, int fmt, int norm, const uint16_t* gamma, const uint16_t* beta,
                        float eps, const float* static_ts, uint8_t* sp_codes, uint8_t* sp_sf, uint8_t* sp_meta,
                        uint8_t* dn_codes, uint8_t* dn_sf, float* ts_out, uint16_t* X_out, uint16_t* X, float* c,
                        float* R, uint8_t* keep) {
  normalize_row(x, K, norm, gamma, beta, eps, X, c);
  if (X_out) memcpy(X_out, X, (size_t)K * 2);
  /* O2 tensor scale (R5) */
  float ts = 1.0f;
  if (fmt == FMT_NVFP4) {
    if (static_ts) ts = *static_ts;
    else {
      uint16_t m = 0;
      for (int64_t k = 0; k < K; ++k) { uint16_t a = X[k] & 0x7FFF; if (a > m) m = a; }
      float a_row = bf16_to_f32(m);
      ts = a_row == 0.0f ? 1.0f : a_row / 2688.0f;
    }
  }
  float inv_ts = 1.0f / ts;
  *ts_out = ts;
  /* O3 mask */
  for (int64_t ch = 0; ch < K / 8; ++ch) {
    int i0, i1;
    top2_pairs(X + ch * 8, &i0, &i1);
    uint8_t nib = (uint8_t)(i0 | (i1 << 2));
    if (ch & 1) sp_meta[ch / 2] |= (uint8_t)(nib << 4); else sp_meta[ch / 2] = nib;
    for (int p = 0; p < 4; ++p) keep[ch * 8 + 2 * p] = keep[ch * 8 + 2 * p + 1] = (p == i0 || p == i1);
  }
  /* O4 backbone + O5 residual, one group of 32 logical k at a time (Eq. 7, Eq. 8) */
  int64_t ns = 0;                                             /* survivors written so far */
  for (int64_t g = 0; g < K / 32; ++g) {
    float a = 0.0f;
    for (int i = 0; i < 32; ++i)
      if (keep[g * 32 + i]) { float v = fabsf(bf16_to_f32(X[g * 32 + i])); if (v > a) a = v; }
    float s_eff, inv;
    block_scale(a, fmt, ts, inv_ts, &sp_sf[g], &s_eff, &inv);
    for (int i = 0; i < 32; ++i) {
      int64_t k = g * 32 + i;
      float xv = bf16_to_f32(X[k]);
      if (!keep[k]) { R[k] = xv; continue; }
      uint8_t code = e2m1_encode(xv * inv);
      float d = e2m1_decode(code) * s_eff;
      R[k] = xv - d;
      if (ns & 1) sp_codes[ns / 2] |= (uint8_t)(code << 4); else sp_codes[ns / 2] = code;
      ++ns;
    }
  }
  /* O6 residual, dense groups */
  int Gd = fmt == FMT_NVFP4 ? 16 : 32;
  for (int64_t g = 0; g < K / Gd; ++g) {
    float a = 0.0f;
    for (int i = 0; i < Gd; ++i) { float v = fabsf(R[g * Gd + i]); if (v > a) a = v; }
    float s_eff, inv;
    block_scale(a, fmt, ts, inv_ts, &dn_sf[g], &s_eff, &inv);
    for (int i = 0; i < Gd; ++i) {
      int64_t k = g * Gd + i;
      uint8_t code = e2m1_encode(R[k] * inv);
      if (k & 1) dn_codes[k / 2] |= (uint8_t)(code << 4); else dn_codes[k / 2] = code;
    }
  }
}

static int pick_threads(int nthreads) {
#ifdef _OPENMP
  return nthreads > 0 ? nthreads : omp_get_max_threads();
#else
  (void)nthreads;
  return 1;
#endif
}

/* Canonical (row-major) outputs: sp_codes [T,K/4], sp_sf [T,K/32], sp_meta [T,K/16], dn_codes [T,K/2],
 * dn_sf [T,K/Gd] (Gd = 16 NVFP4 / 32 MXFP4), ts [T]; X_out [T,K] bf16 bits or NULL.  static_ts NULL = dynamic per-row.
 * Returns the number of threads used, or -1 on a bad argument. */
int so_prepare(const uint16_t* x, int64_t T, int64_t K, int fmt, int norm, const uint16_t* gamma, const uint16_t* beta,
               float eps, const float* static_ts, uint8_t* sp_codes, uint8_t* sp_sf, uint8_t* sp_meta,
               uint8_t* dn_codes, uint8_t* dn_sf, float* ts, uint16_t* X_out, int nthreads) {
  if (K <= 0 || K % 256 || T < 0 || (fmt != FMT_NVFP4 && fmt != FMT_MXFP4) || norm < 0 || norm > 2) return -1;
  if (norm != NORM_NONE && !gamma) return -1;
  int nt = pick_threads(nthreads);
  int64_t Gd = fmt == FMT_NVFP4 ? 16 : 32;
#pragma omp parallel num_threads(nt)
  {
    uint16_t* X = (uint16_t*)malloc((size_t)K * 2);
    float* c = (float*)malloc((size_t)K * 4);
    float* R = (float*)malloc((size_t)K * 4);
    uint8_t* keep = (uint8_t*)malloc((size_t)K);
#pragma omp for schedule(static)
    for (int64_t t = 0; t < T; ++t)
      prepare_row(x + t * K, K, fmt, norm, gamma, beta, eps, static_ts, sp_codes + t * (K / 4), sp_sf + t * (K / 32),
                  sp_meta + t * (K / 16), dn_codes + t * (K / 2), dn_sf + t * (K / Gd), ts + t,
                  X_out ? X_out + t * K : NULL, X, c, R, keep);
    free(X); free(c); free(R); free(keep);
  }
  return nt;
}

/* ---- sharq_quantize_weight (Fig. 2 caption; R7) ---------------------------------------------------- */
/* codes [D,K/2], sf_sp [D,K/32], sf_dn [D,K/16] (NVFP4: every scale twice) or [D,K/32] (MXFP4), ts_w scalar */
int so_quantize_weight(const uint16_t* w, int64_t D, int64_t K, int fmt, uint8_t* codes, uint8_t* sf_sp, uint8_t* sf_dn,
                       float* ts_w, int nthreads) {
  if (K <= 0 || K % 256 || D < 0 || (fmt != FMT_NVFP4 && fmt != FMT_MXFP4)) return -1;
  int nt = pick_threads(nthreads);
  float ts = 1.0f;
  if (fmt == FMT_NVFP4) {
    uint16_t m = 0;
    for (int64_t i = 0; i < D * K; ++i) { uint16_t a = w[i] & 0x7FFF; if (a > m) m = a; }
    float a = bf16_to_f32(m);
    ts = a == 0.0f ? 1.0f : a / 2688.0f;
  }
  float inv_ts = 1.0f / ts;
  *ts_w = ts;
#pragma omp parallel for schedule(static) num_threads(nt)
  for (int64_t d = 0; d < D; ++d) {
    const uint16_t* row = w + d * K;
    for (int64_t g = 0; g < K / 32; ++g) {
      float a = 0.0f;
      for (int i = 0; i < 32; ++i) { float v = fabsf(bf16_to_f32(row[g * 32 + i])); if (v > a) a = v; }
      uint8_t code; float s_eff, inv;
      block_scale(a, fmt, ts, inv_ts, &code, &s_eff, &inv);
      sf_sp[d * (K / 32) + g] = code;
      if (fmt == FMT_NVFP4) sf_dn[d * (K / 16) + 2 * g] = sf_dn[d * (K / 16) + 2 * g + 1] = code;
      else sf_dn[d * (K / 32) + g] = code;
      for (int i = 0; i < 32; ++i) {
        int64_t k = g * 32 + i;
        uint8_t c4 = e2m1_encode(bf16_to_f32(row[k]) * inv);
        if (k & 1) codes[d * (K / 2) + k / 2] |= (uint8_t)(c4 << 4); else codes[d * (K / 2) + k / 2] = c4;
      }
    }
  }
  return nt;
}

/* ---- O7 the linear layer in fp64 (Eq. 9) ------------------------------------------------------------------ */
static inline double sf_value(uint8_t code, int fmt) {
  return fmt == FMT_NVFP4 ? (double)e4m3_decode(code) : (double)e8m0_decode(code);
}

/* Y[i, j] = ( sum_k Asp[rows[i], k] Wsp[cols[j], k] + sum_k Adn[rows[i], k] Wdn[cols[j], k] ) ts[rows[i]] ts_w  in fp64,
 * from the STORED canonical outputs only (what the GEMMs see): the backbone is scattered back to its logical positions
 * through the metadata and read through the weight's sparse (group-32) scale view, the residual through the dense view.
 * rows / cols NULL = all.  Every product code*sf*code*sf is exact in fp64; sums run in ascending k, backbone first. */
int so_linear(int64_t T, int64_t K, int64_t D, int fmt, const uint8_t* sp_codes, const uint8_t* sp_sf,
              const uint8_t* sp_meta, const uint8_t* dn_codes, const uint8_t* dn_sf, const float* ts,
              const uint8_t* w_codes, const uint8_t* w_sf_sp, const uint8_t* w_sf_dn, float ts_w,
              const int64_t* rows, int64_t n_rows, const int64_t* cols, int64_t n_cols, double* Y, int nthreads) {
  if (K <= 0 || K % 256 || (fmt != FMT_NVFP4 && fmt != FMT_MXFP4)) return -1;
  if (!rows) n_rows = T;
  if (!cols) n_cols = D;
  int nt = pick_threads(nthreads);
  int64_t Gd = fmt == FMT_NVFP4 ? 16 : 32;
  double* Asp = (double*)calloc((size_t)(n_rows * K), sizeof(double));
  double* Adn = (double*)malloc((size_t)(n_rows * K) * sizeof(double));
  if (!Asp || !Adn) { free(Asp); free(Adn); return -2; }
#pragma omp parallel for schedule(static) num_threads(nt)
  for (int64_t i = 0; i < n_rows; ++i) {
    int64_t t = rows ? rows[i] : i;
    double* asp = Asp + i * K;
    double* adn = Adn + i * K;
    int64_t ns = 0;
    for (int64_t ch = 0; ch < K / 8; ++ch) {
      uint8_t byte = sp_meta[t * (K / 16) + ch / 2];
      int nib = (ch & 1) ? byte >> 4 : byte & 15;
      int idx[2] = {nib & 3, (nib >> 2) & 3};
      for (int s = 0; s < 2; ++s)
        for (int e = 0; e < 2; ++e) {
          int64_t k = ch * 8 + idx[s] * 2 + e;
          uint8_t b = sp_codes[t * (K / 4) + ns / 2];
          uint8_t code = (ns & 1) ? b >> 4 : b & 15;
          ++ns;
          asp[k] = (double)e2m1_decode(code) * sf_value(sp_sf[t * (K / 32) + k / 32], fmt);
        }
    }
    for (int64_t k = 0; k < K; ++k) {
      uint8_t b = dn_codes[t * (K / 2) + k / 2];
      uint8_t code = (k & 1) ? b >> 4 : b & 15;
      adn[k] = (double)e2m1_decode(code) * sf_value(dn_sf[t * (K / Gd) + k / Gd], fmt);
    }
  }
#pragma omp parallel num_threads(nt)
  {
    double* wsp = (double*)malloc((size_t)K * sizeof(double));
    double* wdn = (double*)malloc((size_t)K * sizeof(double));
#pragma omp for schedule(static)
    for (int64_t j = 0; j < n_cols; ++j) {
      int64_t d = cols ? cols[j] : j;
      for (int64_t k = 0; k < K; ++k) {
        uint8_t b = w_codes[d * (K / 2) + k / 2];
        double v = (double)e2m1_decode((k & 1) ? b >> 4 : b & 15);
        wsp[k] = v * sf_value(w_sf_sp[d * (K / 32) + k / 32], fmt);
        wdn[k] = v * sf_value(w_sf_dn[d * (K / Gd) + k / Gd], fmt);
      }
      for (int64_t i = 0; i < n_rows; ++i) {
        const double* asp = Asp + i * K;
        const double* adn = Adn + i * K;
        double acc = 0.0;
        for (int64_t k = 0; k < K; ++k) acc += asp[k] * wsp[k];
        for (int64_t k = 0; k < K; ++k) acc += adn[k] * wdn[k];
        int64_t t = rows ? rows[i] : i;
        Y[i * n_cols + j] = acc * (double)ts[t] * (double)ts_w;
      }
    }
    free(wsp); free(wdn);
  }
  free(Asp); free(Adn);
  return nt;
}

int so_max_threads(void) { return pick_threads(0); }

/* R1's reduction alone (tests compare it with the numpy oracle on order-sensitive inputs) */
float so_canonical_sum(const float* t, int64_t K, int squares) { return canonical_sum(t, K, squares); }

/* ---- operators folded in front of the preparation (R18) -------------- */
/* h = bf16(x + r): the residual-stream add; the fp32 sum then RNE to bf16 */
void so_residual_add(const uint16_t* x, const uint16_t* r, int64_t n, uint16_t* h) {
  for (int64_t i = 0; i < n; ++i) h[i] = f32_to_bf16(bf16_to_f32(x[i]) + bf16_to_f32(r[i]));
}

/* e ~ exp(-g) by R18's fixed algorithm: every step one binary32 RN operation, no FMA; constants as bit patterns */
static float exp_neg_contract(float g) {
  static const uint32_t kPoly[6] = {0x3F800000u, 0x3F317218u, 0x3E75FDF0u, 0x3D635847u, 0x3C1D955Bu, 0x3AAEC3FFu};  /* RN(ln2^k / k!) */
  const float magic = 12582912.0f;                            /* 1.5 * 2^23 */
  float t = g * bits_f32(0xBFB8AA3Bu);                        /* -RN(log2 e) */
  if (t < -126.0f) t = -126.0f;
  if (t > 126.0f) t = 126.0f;
  volatile float tm = t + magic;                              /* volatile: the compiler must not fold (t + M) - M */
  float n = tm - magic;                                       /* RNE integer of t */
  float f = t - n;
  float p = bits_f32(kPoly[5]);
  for (int k = 4; k >= 0; --k) {
    float pf = p * f;
    p = pf + bits_f32(kPoly[k]);
  }
  return p * bits_f32((uint32_t)((int32_t)n + 127) << 23);    /* p * 2^n */
}

/* h = bf16( silu(g) u ): e = exp_neg(g); den = 1 + e; sig = 1 / den; s = g sig; a = s u; one rounding to bf16 */
void so_swiglu(const uint16_t* gate, const uint16_t* up, int64_t n, uint16_t* h, int nthreads) {
  int nt = pick_threads(nthreads);
#pragma omp parallel for schedule(static) num_threads(nt)
  for (int64_t i = 0; i < n; ++i) {
    float g = bf16_to_f32(gate[i]), u = bf16_to_f32(up[i]);
    float e = exp_neg_contract(g);
    float den = 1.0f + e;
    float sig = 1.0f / den;
    float s = g * sig;
    h[i] = f32_to_bf16(s * u);
  }
}

float so_exp_neg(float g) { return exp_neg_contract(g); }

/* ==== HiF4 (Appendix A.2; R9-R12, R16) ======================================================= */
/* A unit = 64 S1P2 elements + one 32-bit word E6M2 | E1_8 << 8 | E1_16 << 16.  Conversion from BF16 = Algorithm 1
 * (P:496-528), RNE everywhere (R9), BF16 intermediates (R10). */

/* E6M2 (Table 7): value(c) = 2^((c >> 2) - 48) (1 + (c & 3) / 4), codes 0x00 .. 0xFE */
static inline float e6m2_value(int c) { return ldexpf(1.0f + (float)(c & 3) * 0.25f, (c >> 2) - 48); }
/* nearest code, ties to the even mantissa, clamped to [2^-48, 1.5 * 2^15]; by bisection over the monotone grid */
static int e6m2_encode(float sf) {
  if (!(sf >= e6m2_value(0))) return 0;                       /* below the minimum, and 0 (R11) */
  if (sf >= e6m2_value(0xFE)) return 0xFE;
  int lo = 0, hi = 0xFE;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (e6m2_value(mid) <= sf) lo = mid; else hi = mid - 1;
  }
  double dl = (double)sf - (double)e6m2_value(lo), dh = (double)e6m2_value(lo + 1) - (double)sf;
  if (dh < dl || (dh == dl && (lo & 1))) ++lo;
  return lo;
}
/* E6M2_REC_to_BF16: bf16(1 / 1.M) from a 4-entry table, exponent negated */
static inline float e6m2_reciprocal(int c) {
  static const float lut[4] = {1.0f, 0.80078125f, 0.66796875f, 0.5703125f};
  return ldexpf(lut[c & 3], -((c >> 2) - 48));
}
static inline float round_bf16(float x) { return bf16_to_f32(f32_to_bf16(x)); }

/* Algorithm 1 on one unit: V = 64 bf16 bit patterns -> 64 S1P2 codes (bit 3 sign, 3 bits of |.| in quarters) + word */
static void hif4_encode_unit(const uint16_t* V, uint8_t* codes, uint32_t* word) {
  float v16[16], v8[8], vmax = 0.0f;
  for (int j = 0; j < 16; ++j) {                              /* stage 1: three-level tree of maxima (lines 1-8) */
    float m = 0.0f;
    for (int i = 0; i < 4; ++i) { float a = fabsf(bf16_to_f32(V[4 * j + i])); if (a > m) m = a; }
    v16[j] = m;
  }
  for (int g = 0; g < 8; ++g) { v8[g] = v16[2 * g] > v16[2 * g + 1] ? v16[2 * g] : v16[2 * g + 1]; if (v8[g] > vmax) vmax = v8[g]; }
  float sf = round_bf16(vmax * 0.142578125f);                 /* line 10: (1/7) in bf16, bf16 multiply */
  int e6 = e6m2_encode(sf);                                   /* line 11 */
  float rec = e6m2_reciprocal(e6);                            /* line 12 */
  uint32_t w = (uint32_t)e6;
  float s8[8], s16[16];
  for (int g = 0; g < 8; ++g) {                               /* line 13 */
    int b = v8[g] * rec >= 4.0f;
    s8[g] = b ? 0.5f : 1.0f;
    w |= (uint32_t)b << (8 + g);
  }
  for (int j = 0; j < 16; ++j) {                              /* line 14 */
    int b = (v16[j] * rec) * s8[j / 2] >= 2.0f;
    s16[j] = b ? 0.5f : 1.0f;
    w |= (uint32_t)b << (16 + j);
  }
  for (int i = 0; i < 64; ++i) {                              /* lines 17-21: scale (a BF16 value, R10), then S1P2 */
    float scaled = (round_bf16(bf16_to_f32(V[i]) * rec) * s8[i / 8]) * s16[i / 4];
    float q = nearbyintf(fabsf(scaled) * 4.0f);               /* RNE (default rounding mode) */
    int mag = q > 7.0f ? 7 : (int)q;
    codes[i] = (uint8_t)(mag | ((f32_bits(scaled) >> 31) << 3));
  }
  *word = w;
}
/* Eq. 15, 0-based integer division (R16): V_i = E6M2 2^(E1_8[i / 8] + E1_16[i / 4]) S1P2_i; exact in fp32 */
static inline float hif4_decode(uint8_t code, uint32_t word, int i) {
  float mag = (float)(code & 7) * 0.25f;
  int sh = (int)((word >> (8 + i / 8)) & 1u) + (int)((word >> (16 + i / 4)) & 1u);
  float v = ldexpf(mag, sh) * e6m2_value((int)(word & 0xFFu));
  return (code & 8) ? -v : v;
}

/* 2:4: the two largest |x| of four, ties to the lower index */
static void top2_of4(const uint16_t* X4, int* i0, int* i1) {
  int first = 0, second = -1;
  for (int p = 1; p < 4; ++p) if ((X4[p] & 0x7FFF) > (X4[first] & 0x7FFF)) first = p;
  for (int p = 0; p < 4; ++p) {
    if (p == first) continue;
    if (second < 0 || (X4[p] & 0x7FFF) > (X4[second] & 0x7FFF)) second = p;
  }
  *i0 = first < second ? first : second;
  *i1 = first < second ? second : first;
}

/* sharq_prepare with HiF4: sp_codes [T,K/4], sp_sf u32 [T,K/64], sp_meta [T,K/8] (one nibble per 4 elements),
 * dn_codes [T,K/2], dn_sf u32 [T,K/64]; ts = 1 */
int so_prepare_hif4(const uint16_t* x, int64_t T, int64_t K, int norm, const uint16_t* gamma, const uint16_t* beta,
                    float eps, uint8_t* sp_codes, uint32_t* sp_sf, uint8_t* sp_meta, uint8_t* dn_codes, uint32_t* dn_sf,
                    int nthreads) {
  if (K <= 0 || K % 256 || T < 0 || norm < 0 || norm > 2 || (norm != NORM_NONE && !gamma)) return -1;
  int nt = pick_threads(nthreads);
#pragma omp parallel num_threads(nt)
  {
    uint16_t* X = (uint16_t*)malloc((size_t)K * 2);
    uint16_t* Xsp = (uint16_t*)malloc((size_t)K * 2);
    uint16_t* Rb = (uint16_t*)malloc((size_t)K * 2);
    float* c = (float*)malloc((size_t)K * 4);
    uint8_t* keep = (uint8_t*)malloc((size_t)K);
    uint8_t* code = (uint8_t*)malloc((size_t)K);
#pragma omp for schedule(static)
    for (int64_t t = 0; t < T; ++t) {
      normalize_row(x + t * K, K, norm, gamma, beta, eps, X, c);
      for (int64_t q = 0; q < K / 4; ++q) {                   /* mask; M (.) X has +0 at dropped positions */
        int i0, i1;
        top2_of4(X + 4 * q, &i0, &i1);
        uint8_t nib = (uint8_t)(i0 | (i1 << 2));
        uint8_t* m = sp_meta + t * (K / 8) + q / 2;
        if (q & 1) *m |= (uint8_t)(nib << 4); else *m = nib;
        for (int p = 0; p < 4; ++p) { keep[4 * q + p] = (p == i0 || p == i1); Xsp[4 * q + p] = keep[4 * q + p] ? X[4 * q + p] : 0; }
      }
      int64_t ns = 0;
      for (int64_t u = 0; u < K / 64; ++u) {                  /* backbone: Alg. 1 on 64 LOGICAL positions (R12) */
        uint32_t w;
        hif4_encode_unit(Xsp + 64 * u, code + 64 * u, &w);
        sp_sf[t * (K / 64) + u] = w;
        for (int i = 0; i < 64; ++i) {
          int64_t k = 64 * u + i;
          float xf = bf16_to_f32(X[k]);
          float r = xf;
          if (keep[k]) {
            r = xf - hif4_decode(code[k], w, i);              /* Eq. 8 */
            uint8_t* dst = sp_codes + t * (K / 4) + ns / 2;
            if (ns & 1) *dst |= (uint8_t)(code[k] << 4); else *dst = code[k];
            ++ns;
          }
          Rb[k] = f32_to_bf16(r);                             /* Alg. 1 takes BF16 input */
        }
      }
      for (int64_t u = 0; u < K / 64; ++u) {                  /* residual */
        uint32_t w;
        hif4_encode_unit(Rb + 64 * u, code + 64 * u, &w);
        dn_sf[t * (K / 64) + u] = w;
        for (int i = 0; i < 64; i += 2) dn_codes[t * (K / 2) + (64 * u + i) / 2] = (uint8_t)(code[64 * u + i] | (code[64 * u + i + 1] << 4));
      }
    }
    free(X); free(Xsp); free(Rb); free(c); free(keep); free(code);
  }
  return nt;
}

int so_quantize_weight_hif4(const uint16_t* w, int64_t D, int64_t K, uint8_t* codes, uint32_t* sf, int nthreads) {
  if (K <= 0 || K % 256 || D < 0) return -1;
  int nt = pick_threads(nthreads);
#pragma omp parallel for schedule(static) num_threads(nt)
  for (int64_t d = 0; d < D; ++d)
    for (int64_t u = 0; u < K / 64; ++u) {
      uint8_t c[64];
      hif4_encode_unit(w + d * K + 64 * u, c, &sf[d * (K / 64) + u]);
      for (int i = 0; i < 64; i += 2) codes[d * (K / 2) + (64 * u + i) / 2] = (uint8_t)(c[i] | (c[i + 1] << 4));
    }
  return nt;
}

/* Eq. 9 in fp64 for HiF4 from the stored arrays (backbone scattered through the 2:4 metadata) */
int so_linear_hif4(int64_t T, int64_t K, int64_t D, const uint8_t* sp_codes, const uint32_t* sp_sf, const uint8_t* sp_meta,
                   const uint8_t* dn_codes, const uint32_t* dn_sf, const uint8_t* w_codes, const uint32_t* w_sf,
                   const int64_t* rows, int64_t n_rows, const int64_t* cols, int64_t n_cols, double* Y, int nthreads) {
  if (K <= 0 || K % 256) return -1;
  if (!rows) n_rows = T;
  if (!cols) n_cols = D;
  int nt = pick_threads(nthreads);
  double* A = (double*)calloc((size_t)(n_rows * K), sizeof(double));     /* backbone at its logical positions, 0 elsewhere */
  double* B = (double*)malloc((size_t)(n_rows * K) * sizeof(double));     /* residual */
  if (!A || !B) { free(A); free(B); return -2; }
#pragma omp parallel for schedule(static) num_threads(nt)
  for (int64_t i = 0; i < n_rows; ++i) {
    int64_t t = rows ? rows[i] : i, ns = 0;
    for (int64_t q = 0; q < K / 4; ++q) {
      uint8_t byte = sp_meta[t * (K / 8) + q / 2];
      int nib = (q & 1) ? byte >> 4 : byte & 15;
      int idx[2] = {nib & 3, (nib >> 2) & 3};
      for (int s = 0; s < 2; ++s) {
        int64_t k = 4 * q + idx[s];
        uint8_t b = sp_codes[t * (K / 4) + ns / 2];
        uint8_t code = (ns & 1) ? b >> 4 : b & 15;
        ++ns;
        A[i * K + k] = (double)hif4_decode(code, sp_sf[t * (K / 64) + k / 64], (int)(k % 64));
      }
    }
    for (int64_t k = 0; k < K; ++k) {
      uint8_t b = dn_codes[t * (K / 2) + k / 2];
      B[i * K + k] = (double)hif4_decode((k & 1) ? b >> 4 : b & 15, dn_sf[t * (K / 64) + k / 64], (int)(k % 64));
    }
  }
#pragma omp parallel num_threads(nt)
  {
    double* wv = (double*)malloc((size_t)K * sizeof(double));
#pragma omp for schedule(static)
    for (int64_t j = 0; j < n_cols; ++j) {
      int64_t d = cols ? cols[j] : j;
      for (int64_t k = 0; k < K; ++k) {
        uint8_t b = w_codes[d * (K / 2) + k / 2];
        wv[k] = (double)hif4_decode((k & 1) ? b >> 4 : b & 15, w_sf[d * (K / 64) + k / 64], (int)(k % 64));
      }
      for (int64_t i = 0; i < n_rows; ++i) {
        double acc = 0.0;
        for (int64_t k = 0; k < K; ++k) acc += A[i * K + k] * wv[k];
        for (int64_t k = 0; k < K; ++k) acc += B[i * K + k] * wv[k];
        Y[i * n_cols + j] = acc;
      }
    }
    free(wv);
  }
  free(A); free(B);
  return nt;
}
