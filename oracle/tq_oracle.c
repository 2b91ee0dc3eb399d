/*
 * tq_oracle.c — CPU ORACLE for the TurboESM hot path (arxiv/paper_2603_26110).  TEST INFRASTRUCTURE.
 *
 * This file is the parity oracle: a plain, slow, step-by-step restatement of what the paper and
 * BASELINE.json:north_star define, in fp64.  It shares no code, header, table or constant with the CUDA
 * product under paper_2603_26110_b200/csrc and must never be imported, linked or executed by the
 * product path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may use it.
 *
 * Order and notation follow the paper:
 *   RoPE                       PAPER.md:47-56  (Eq. 1-2), pair convention PAPER.md:102
 *   RoPE-first PI rotation     PAPER.md:104-116 (Eq. 4, prefill steps 1,3,4)
 *   Lloyd-Max 8-level coding   PAPER.md:145-152 (Eq. 5), dual K/V LUT PAPER.md:154-164, argmin PAPER.md:217
 *   residual sign sketch       PAPER.md:166-179 (Eq. 6-7), generalised to sign(S r) and a stored |r|
 *                              as BASELINE.json:north_star requires (reading D2)
 *   packing                    PAPER.md:199-213 (8 codes at shifts 0,3,..,21), 3 bytes per 8 codes (D5)
 *   decode                     PAPER.md:118-124 and Algorithm 1, two-pass exact softmax
 *   paper-literal Eq. 6-7 mode PAPER.md:166-179 as printed (tqo_quantize_vector_literal / _pack_literal)
 *   V-side residual sketch     Algorithm 1 line 10, PAPER.md:234 (tqo_value_sketch_planes / tqo_decode_attn_vq)
 *
 * Pins (tests/test_oracle_*.py): every function below is checked against something other than itself —
 * closed forms, textbook tables, numpy library routines, brute force, Monte-Carlo.  Parity unpinned: none
 * of the arithmetic; the only unpinned quantity is the *reported* cosine against unquantised attention
 * (tqo_dense_attn_ref is pinned, the paper's >0.96 figure is not reproducible here — see DESIGN.md).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TQO_PI 3.14159265358979323846

int tqo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void tqo_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ---- IEEE binary16 <-> fp64, written out (pinned against numpy.float16 in the tests) -------------- */

/* fp64 -> binary16 bits, round-to-nearest-even, finite inputs >= 0 clamped to 65504 (D6). */
uint16_t tqo_f64_to_f16(double x) {
  uint16_t sign = 0;
  if (x < 0) {
    sign = 0x8000;
    x = -x;
  }
  if (x != x) return (uint16_t)(sign | 0x7e00);
  if (x >= 65504.0) return (uint16_t)(sign | 0x7bff); /* clamp, never inf */
  if (x == 0.0) return sign;
  int e;
  double f = frexp(x, &e); /* x = f * 2^e, f in [0.5, 1) */
  /* normal binary16: x = 1.m * 2^(E-15), E in [1,30]; smallest normal 2^-14 */
  int E = e - 1 + 15;
  double scaled;
  if (E >= 1) {
    /* mantissa steps of 2^(e-1-10) */
    scaled = ldexp(x, 10 - (e - 1)); /* in [1024, 2048) */
  } else {
    /* subnormal: steps of 2^-24 */
    scaled = ldexp(x, 24);
    E = 0;
  }
  (void)f;
  double fl = floor(scaled);
  double rem = scaled - fl;
  uint32_t q = (uint32_t)fl;
  if (rem > 0.5 || (rem == 0.5 && (q & 1u))) q += 1;
  uint32_t bits;
  if (E >= 1) {
    /* q in [1024, 2048]; 2048 means carry into the exponent */
    bits = ((uint32_t)E << 10) + (q - 1024u);
  } else {
    bits = q; /* q == 1024 becomes the smallest normal automatically */
  }
  if (bits > 0x7bffu) bits = 0x7bffu;
  return (uint16_t)(sign | bits);
}

double tqo_f16_to_f64(uint16_t h) {
  int sign = (h >> 15) & 1;
  int E = (h >> 10) & 0x1f;
  int m = h & 0x3ff;
  double v;
  if (E == 0)
    v = ldexp((double)m, -24);
  else if (E == 31)
    v = m ? NAN : INFINITY;
  else
    v = ldexp(1.0 + (double)m / 1024.0, E - 15);
  return sign ? -v : v;
}

/* ---- RoPE, Eq. 1-2 ---------------------------------------------------------------
 * theta_g = base^(-2g/d), g = 0..d/2-1.  layout 0: pairs (2g, 2g+1); layout 1: (g, g+d/2).
 * (x_a, x_b) -> (x_a cos(p theta) - x_b sin(p theta), x_a sin(p theta) + x_b cos(p theta)).             */
void tqo_rope(const double *x, int d, double pos, double base, int layout, double *out) {
  for (int g = 0; g < d / 2; ++g) {
    double theta = pow(base, -2.0 * (double)g / (double)d);
    double c = cos(pos * theta), s = sin(pos * theta);
    int a = layout == 0 ? 2 * g : g;
    int b = layout == 0 ? 2 * g + 1 : g + d / 2;
    out[a] = x[a] * c - x[b] * s;
    out[b] = x[a] * s + x[b] * c;
  }
}

/* y = M x, M row-major (rows x cols) given in fp32, widened exactly. */
static void matvec_f32(const float *M, int rows, int cols, const double *x, double *y) {
  for (int i = 0; i < rows; ++i) {
    double acc = 0.0;
    for (int k = 0; k < cols; ++k) acc += (double)M[(size_t)i * cols + k] * x[k];
    y[i] = acc;
  }
}

/* y = M^T x */
static void matvec_t_f32(const float *M, int rows, int cols, const double *x, double *y) {
  for (int k = 0; k < cols; ++k) y[k] = 0.0;
  for (int i = 0; i < rows; ++i)
    for (int k = 0; k < cols; ++k) y[k] += (double)M[(size_t)i * cols + k] * x[i];
}

/* ---- Lloyd-Max coding, Eq. 5 ---------------------------------------------------
 * Decision thresholds are the centroid midpoints evaluated in fp32 (t_k = 0.5f*(c_k + c_{k+1})), so both
 * implementations hold bit-identical thresholds (D7); the comparison itself is done on the
 * fp64 coordinate.  code = #{k : u > t_k}; a coordinate exactly on a threshold takes the lower code,
 * which is what a first-minimum argmin over the LUT returns.                            */
int tqo_code(double u, const float *lut8) {
  int code = 0;
  for (int k = 0; k < 7; ++k) {
    float t = 0.5f * (lut8[k] + lut8[k + 1]);
    if (u > (double)t) code += 1;
  }
  return code;
}

/* Brute-force nearest centroid (first minimum), used by the tests to pin tqo_code. */
int tqo_code_argmin(double u, const float *lut8) {
  int best = 0;
  double bd = fabs(u - (double)lut8[0]);
  for (int k = 1; k < 8; ++k) {
    double dk = fabs(u - (double)lut8[k]);
    if (dk < bd) {
      bd = dk;
      best = k;
    }
  }
  return best;
}

/* ---- packing, PAPER.md:203-213 --------------------------------------------------------------------
 * The paper packs 8 indices per INT32: packed = sum_i idx_i << (3 i).  The canonical stream keeps the low
 * 24 bits of that container as 3 little-endian bytes (D5).                                             */
void tqo_pack_codes(const uint8_t *codes, int d, uint8_t *out) {
  for (int grp = 0; grp < d / 8; ++grp) {
    uint32_t packed = 0;
    for (int i = 0; i < 8; ++i) packed += (uint32_t)codes[8 * grp + i] << (3 * i);
    out[3 * grp + 0] = (uint8_t)(packed & 0xff);
    out[3 * grp + 1] = (uint8_t)((packed >> 8) & 0xff);
    out[3 * grp + 2] = (uint8_t)((packed >> 16) & 0xff);
  }
}

void tqo_unpack_codes(const uint8_t *in, int d, uint8_t *codes) {
  for (int grp = 0; grp < d / 8; ++grp) {
    uint32_t packed = (uint32_t)in[3 * grp] | ((uint32_t)in[3 * grp + 1] << 8) | ((uint32_t)in[3 * grp + 2] << 16);
    for (int i = 0; i < 8; ++i) codes[8 * grp + i] = (uint8_t)((packed >> (3 * i)) & 0x7);
  }
}

void tqo_pack_bits(const uint8_t *bits, int m, uint8_t *out) {
  for (int byte = 0; byte < m / 8; ++byte) {
    unsigned v = 0;
    for (int j = 0; j < 8; ++j) v |= (unsigned)(bits[8 * byte + j] & 1) << j;
    out[byte] = (uint8_t)v;
  }
}

void tqo_unpack_bits(const uint8_t *in, int m, uint8_t *bits) {
  for (int j = 0; j < m; ++j) bits[j] = (uint8_t)((in[j / 8] >> (j % 8)) & 1);
}

/* ---- quantize one vector (steps 1-5 of DESIGN.md "oracle: quantize") -------------------------------
 * x[d]: the vector widened to fp64.  is_key: apply RoPE at `pos` and build the residual sketch.
 * Outputs: codes[d]; bits[m] and *rnorm_h (keys only); *norm_h; optionally u_out[d] (unit vector) for the
 * near-threshold diagnostics.                                                                          */
void tqo_quantize_vector(const double *x, int d, int m, int is_key, double pos, double base, int layout,
                         const float *Pi, const float *lut8, const float *S, uint8_t *codes, uint8_t *bits,
                         uint16_t *norm_h, uint16_t *rnorm_h, double *u_out) {
  double xr[256], y[256], u[256], r[256], sr[256];
  if (is_key)
    tqo_rope(x, d, pos, base, layout, xr); /* step 1: x' = R x */
  else
    memcpy(xr, x, sizeof(double) * (size_t)d);
  matvec_f32(Pi, d, d, xr, y); /* step 2: y = PI x' */
  double n2 = 0.0;
  for (int i = 0; i < d; ++i) n2 += y[i] * y[i];
  double n = sqrt(n2); /* step 3: norm               (north_star)   */
  for (int i = 0; i < d; ++i) u[i] = n > 0.0 ? y[i] / n : 0.0;
  *norm_h = tqo_f64_to_f16(n);
  for (int i = 0; i < d; ++i) codes[i] = (uint8_t)tqo_code(u[i], lut8); /* step 4: Eq. 5 */
  if (u_out) memcpy(u_out, u, sizeof(double) * (size_t)d);
  if (is_key) { /* step 5: r = u - lut[code]; |r|; sign(S r)   (Eq. 6 generalised, D2) */
    double g2 = 0.0;
    for (int i = 0; i < d; ++i) {
      r[i] = u[i] - (double)lut8[codes[i]];
      g2 += r[i] * r[i];
    }
    *rnorm_h = tqo_f64_to_f16(sqrt(g2));
    matvec_f32(S, m, d, r, sr);
    for (int j = 0; j < m; ++j) bits[j] = (uint8_t)(sr[j] >= 0.0 ? 1 : 0); /* tie: >= 0 -> 1 (D7) */
  }
}

/* ---- quantize-and-pack over one layer -----------------------------------------------------------
 * k, v: [B][H][T][d] fp32 (fp16 inputs are widened exactly by the caller).  Token i has cache index and
 * RoPE position start_pos + i.  pi_k/pi_v: [H][d][d] of this layer, lut_k/lut_v: [H][8], S: [m][d].
 * Canonical planes indexed [b][h][t].  near_k/near_v (optional, [b][h][t][d] bytes): 1 where the unit
 * coordinate lies within near_eps of a decision threshold (the tolerance band of north_star).
 * amb_sign (optional, [b][h][t][m]): 1 where |(S r)_j| < sign_eps.                                      */
void tqo_quantize_pack(int B, int H, int T, int d, int m, double base, int layout, int start_pos,
                       const float *k, const float *v, const float *pi_k, const float *pi_v,
                       const float *lut_k, const float *lut_v, const float *S, uint8_t *k_codes,
                       uint8_t *k_signs, uint16_t *k_norm, uint16_t *k_rnorm, uint8_t *v_codes,
                       uint16_t *v_norm, double near_eps, uint8_t *near_k, uint8_t *near_v) {
  const int cb = 3 * d / 8, sb = m / 8;
  long total = (long)B * H * T;
#pragma omp parallel for schedule(static)
  for (long idx = 0; idx < total; ++idx) {
    int t = (int)(idx % T);
    int h = (int)((idx / T) % H);
    double x[256], u[256];
    uint8_t codes[256], bits[256];
    uint16_t nh = 0, rh = 0;
    const float *kp = k + (size_t)idx * d;
    const float *vp = v + (size_t)idx * d;
    const float *luk = lut_k + (size_t)h * 8, *luv = lut_v + (size_t)h * 8;
    /* key */
    for (int i = 0; i < d; ++i) x[i] = (double)kp[i];
    tqo_quantize_vector(x, d, m, 1, (double)(start_pos + t), base, layout, pi_k + (size_t)h * d * d, luk, S,
                        codes, bits, &nh, &rh, u);
    tqo_pack_codes(codes, d, k_codes + (size_t)idx * cb);
    tqo_pack_bits(bits, m, k_signs + (size_t)idx * sb);
    k_norm[idx] = nh;
    k_rnorm[idx] = rh;
    if (near_k)
      for (int i = 0; i < d; ++i) {
        uint8_t nr = 0;
        for (int q = 0; q < 7; ++q) {
          float th = 0.5f * (luk[q] + luk[q + 1]);
          if (fabs(u[i] - (double)th) < near_eps) nr = 1;
        }
        near_k[(size_t)idx * d + i] = nr;
      }
    /* value: no RoPE, no sketch (D3) */
    for (int i = 0; i < d; ++i) x[i] = (double)vp[i];
    tqo_quantize_vector(x, d, m, 0, 0.0, base, layout, pi_v + (size_t)h * d * d, luv, S, codes, bits, &nh, &rh,
                        u);
    tqo_pack_codes(codes, d, v_codes + (size_t)idx * cb);
    v_norm[idx] = nh;
    if (near_v)
      for (int i = 0; i < d; ++i) {
        uint8_t nr = 0;
        for (int q = 0; q < 7; ++q) {
          float th = 0.5f * (luv[q] + luv[q + 1]);
          if (fabs(u[i] - (double)th) < near_eps) nr = 1;
        }
        near_v[(size_t)idx * d + i] = nr;
      }
  }
}

/* ---- paper-literal residual correction, Eq. 6-7 as printed ---------
 * The paper stores s = sign(x - x^) per coordinate (Eq. 6) and reconstructs x~ = x^ + s e-bar with ONE pre-calibrated
 * scalar e-bar per head (Eq. 7); its LUT is calibrated on the rotated activations themselves (no norm is stored,
 * PAPER.md:159-164) and V is not rotated (PAPER.md:157, 162 — PI_V = I is passed as data).  In the canonical planes
 * this is: codes on y = PI x' (no normalisation), norm plane = 1.0, bits_j = [(S e)_j >= 0] with e = y - lut[code]
 * (S = I as data gives Eq. 6's sign(e_j)), and the rnorm plane = binary16(e-bar m sqrt(2/pi)), so that the decode
 * correction  sqrt(pi/2)/m * rnorm * <S q'', sigma>  of tqo_decode_attn equals  e-bar <q'', s>  — Eq. 7 contracted
 * with the query (Algorithm 1 line 6).  y_out (optional): the coded coordinates.                     */
void tqo_quantize_vector_literal(const double *x, int d, int m, int is_key, double pos, double base, int layout,
                                 const float *Pi, const float *lut8, const float *S, double ebar, uint8_t *codes,
                                 uint8_t *bits, uint16_t *norm_h, uint16_t *rnorm_h, double *y_out) {
  double xr[256], y[256], e[256], se[256];
  if (is_key)
    tqo_rope(x, d, pos, base, layout, xr);
  else
    memcpy(xr, x, sizeof(double) * (size_t)d);
  matvec_f32(Pi, d, d, xr, y);
  *norm_h = tqo_f64_to_f16(1.0);
  for (int i = 0; i < d; ++i) codes[i] = (uint8_t)tqo_code(y[i], lut8); /* Eq. 5 on the activation itself */
  if (y_out) memcpy(y_out, y, sizeof(double) * (size_t)d);
  if (is_key) {
    for (int i = 0; i < d; ++i) e[i] = y[i] - (double)lut8[codes[i]];  /* e = x - x^                 (Eq. 6) */
    matvec_f32(S, m, d, e, se);
    for (int j = 0; j < m; ++j) bits[j] = (uint8_t)(se[j] >= 0.0 ? 1 : 0);
    *rnorm_h = tqo_f64_to_f16(ebar * (double)m * sqrt(2.0 / TQO_PI)); /* e-bar, in the units of the rnorm plane */
  }
}

/* Layer form of the above; same conventions as tqo_quantize_pack.  ebar_k: [H].  near_k / near_v: 1 where the coded
 * coordinate lies within near_eps * max(1, |y|_2) of a decision threshold (the band scales with the vector here,
 * because the coordinates are not normalised).                                                                  */
void tqo_quantize_pack_literal(int B, int H, int T, int d, int m, double base, int layout, int start_pos,
                               const float *k, const float *v, const float *pi_k, const float *pi_v,
                               const float *lut_k, const float *lut_v, const float *S, const float *ebar_k,
                               uint8_t *k_codes, uint8_t *k_signs, uint16_t *k_norm, uint16_t *k_rnorm,
                               uint8_t *v_codes, uint16_t *v_norm, double near_eps, uint8_t *near_k, uint8_t *near_v) {
  const int cb = 3 * d / 8, sb = m / 8;
  long total = (long)B * H * T;
#pragma omp parallel for schedule(static)
  for (long idx = 0; idx < total; ++idx) {
    int t = (int)(idx % T);
    int h = (int)((idx / T) % H);
    double x[256], y[256];
    uint8_t codes[256], bits[256];
    uint16_t nh = 0, rh = 0;
    for (int side = 0; side < 2; ++side) {
      const float *xp = (side == 0 ? k : v) + (size_t)idx * d;
      const float *lu = (side == 0 ? lut_k : lut_v) + (size_t)h * 8;
      for (int i = 0; i < d; ++i) x[i] = (double)xp[i];
      tqo_quantize_vector_literal(x, d, m, side == 0, (double)(start_pos + t), base, layout,
                                  (side == 0 ? pi_k : pi_v) + (size_t)h * d * d, lu, S, side == 0 ? (double)ebar_k[h] : 0.0,
                                  codes, bits, &nh, &rh, y);
      tqo_pack_codes(codes, d, (side == 0 ? k_codes : v_codes) + (size_t)idx * cb);
      if (side == 0) {
        tqo_pack_bits(bits, m, k_signs + (size_t)idx * sb);
        k_norm[idx] = nh;
        k_rnorm[idx] = rh;
      } else {
        v_norm[idx] = nh;
      }
      uint8_t *near = side == 0 ? near_k : near_v;
      if (near) {
        double n2 = 0.0;
        for (int i = 0; i < d; ++i) n2 += y[i] * y[i];
        double band = near_eps * fmax(1.0, sqrt(n2));
        for (int i = 0; i < d; ++i) {
          uint8_t nr = 0;
          for (int q = 0; q < 7; ++q) {
            float th = 0.5f * (lu[q] + lu[q + 1]);
            if (fabs(y[i] - (double)th) < band) nr = 1;
          }
          near[(size_t)idx * d + i] = nr;
        }
      }
    }
  }
}

/* (S r)_j for one key vector, so a test can skip sign bits whose pre-image is within rounding of 0. */
void tqo_key_sketch_values(const float *kvec, int d, int m, double pos, double base, int layout,
                           const float *Pi, const float *lut8, const float *S, double *sr_out) {
  double x[256], xr[256], y[256], r[256];
  for (int i = 0; i < d; ++i) x[i] = (double)kvec[i];
  tqo_rope(x, d, pos, base, layout, xr);
  matvec_f32(Pi, d, d, xr, y);
  double n2 = 0.0;
  for (int i = 0; i < d; ++i) n2 += y[i] * y[i];
  double n = sqrt(n2);
  for (int i = 0; i < d; ++i) {
    double u = n > 0.0 ? y[i] / n : 0.0;
    r[i] = u - (double)lut8[tqo_code(u, lut8)];
  }
  matvec_f32(S, m, d, r, sr_out);
}

/* ---- decode attention over one layer's canonical planes (steps 7-10) -------------------------------
 * q: [B][H][d] fp32 pre-RoPE; q_pos[b]: RoPE position of the query; seq_len[b]: tokens attended.
 * planes indexed [b][h][t] with row stride T_stride tokens.  out: [B][H][d] fp64.
 *   q'' = PI_K RoPE(q, p_q);  z = S q''                                   (Eq. 4; north_star)
 *   s_j = n_j ( <q'', lut_K[code_j]> + sqrt(pi/2)/m * g_j <z, sigma_j> ) / sqrt(d)   (Alg. 1 l.6-8; D2)
 *   p = softmax(s)  (two-pass, exact)                                     (Alg. 1 l.9)
 *   o' = sum_j p_j nv_j lut_V[codeV_j];  out = PI_V^T o'                   (Alg. 1 l.10-13; north_star)
 * use_qjl = 0 drops the correction term (ablation).                                      */
void tqo_decode_attn(int B, int H, int d, int m, int T_stride, double base, int layout, const float *q,
                     const int32_t *q_pos, const int32_t *seq_len, const float *pi_k, const float *pi_v,
                     const float *lut_k, const float *lut_v, const float *S, const uint8_t *k_codes,
                     const uint8_t *k_signs, const uint16_t *k_norm, const uint16_t *k_rnorm,
                     const uint8_t *v_codes, const uint16_t *v_norm, int use_qjl, double *out) {
  const int cb = 3 * d / 8, sb = m / 8;
  const double cq = sqrt(TQO_PI / 2.0) / (double)m;
#pragma omp parallel for schedule(dynamic)
  for (int unit = 0; unit < B * H; ++unit) {
    int b = unit / H, h = unit % H;
    int T = seq_len[b];
    double qv[256], qr[256], q2[256], z[256], o[256];
    for (int i = 0; i < d; ++i) qv[i] = (double)q[(size_t)unit * d + i];
    tqo_rope(qv, d, (double)q_pos[b], base, layout, qr);
    matvec_f32(pi_k + (size_t)h * d * d, d, d, qr, q2);
    matvec_f32(S, m, d, q2, z);
    const float *luk = lut_k + (size_t)h * 8, *luv = lut_v + (size_t)h * 8;
    double *s = (double *)malloc(sizeof(double) * (size_t)(T > 0 ? T : 1));
    uint8_t codes[256], bits[256];
    double smax = -INFINITY;
    for (int j = 0; j < T; ++j) {
      size_t e = (size_t)unit * T_stride + j;
      tqo_unpack_codes(k_codes + e * cb, d, codes);
      tqo_unpack_bits(k_signs + e * sb, m, bits);
      double a = 0.0, bq = 0.0;
      for (int i = 0; i < d; ++i) a += q2[i] * (double)luk[codes[i]];
      for (int i = 0; i < m; ++i) bq += z[i] * (bits[i] ? 1.0 : -1.0);
      double n = tqo_f16_to_f64(k_norm[e]), g = tqo_f16_to_f64(k_rnorm[e]);
      double corr = use_qjl ? cq * g * bq : 0.0;
      s[j] = n * (a + corr) / sqrt((double)d);
      if (s[j] > smax) smax = s[j];
    }
    double l = 0.0;
    for (int i = 0; i < d; ++i) o[i] = 0.0;
    for (int j = 0; j < T; ++j) {
      size_t e = (size_t)unit * T_stride + j;
      double p = exp(s[j] - smax);
      l += p;
      tqo_unpack_codes(v_codes + e * cb, d, codes);
      double nv = tqo_f16_to_f64(v_norm[e]);
      for (int i = 0; i < d; ++i) o[i] += p * nv * (double)luv[codes[i]];
    }
    for (int i = 0; i < d; ++i) o[i] = T > 0 ? o[i] / l : 0.0;
    matvec_t_f32(pi_v + (size_t)h * d * d, d, d, o, out + (size_t)unit * d);
    free(s);
  }
}

/* ---- V-side residual sketch (Algorithm 1 line 10, "v = LUT_V[idx_v] + sign_v * e_v"; SURVEY.md 8(f)
 * NEXT-1, 8(c) step 10; reading D3: tq_shape.v_qjl = 1) ------------------------------------------------
 * Values get the same treatment as keys minus RoPE: y = PI_V v, n = |y|, u = y / n, codes on u, r = u - lut_V[code],
 * bits_j = [(S r)_j >= 0], rnorm = |r|.  A dequantised value is then the JL reconstruction
 *   v~ = n ( lut_V[code] + sqrt(pi/2)/m * |r| * S^T sigma ),  sigma = 2 bits - 1,
 * whose inner product with any vector is the estimator of tqo_qjl_estimate (E over S of the second term = r).
 * This function only adds the two value planes; codes and norms are those of tqo_quantize_pack.                   */
void tqo_value_sketch_planes(int B, int H, int T, int d, int m, const float *v, const float *pi_v, const float *lut_v,
                             const float *S, uint8_t *v_signs, uint16_t *v_rnorm) {
  const int sb = m / 8;
  long total = (long)B * H * T;
#pragma omp parallel for schedule(static)
  for (long idx = 0; idx < total; ++idx) {
    int h = (int)((idx / T) % H);
    double x[256], y[256], r[256], sr[256];
    uint8_t bits[256];
    const float *lu = lut_v + (size_t)h * 8;
    for (int i = 0; i < d; ++i) x[i] = (double)v[(size_t)idx * d + i];
    matvec_f32(pi_v + (size_t)h * d * d, d, d, x, y);
    double n2 = 0.0, g2 = 0.0;
    for (int i = 0; i < d; ++i) n2 += y[i] * y[i];
    double n = sqrt(n2);
    for (int i = 0; i < d; ++i) {
      double u = n > 0.0 ? y[i] / n : 0.0;
      r[i] = u - (double)lu[tqo_code(u, lu)];
      g2 += r[i] * r[i];
    }
    matvec_f32(S, m, d, r, sr);
    for (int j = 0; j < m; ++j) bits[j] = (uint8_t)(sr[j] >= 0.0 ? 1 : 0);
    tqo_pack_bits(bits, m, v_signs + (size_t)idx * sb);
    v_rnorm[idx] = tqo_f64_to_f16(sqrt(g2));
  }
}

/* Decode attention with the V-side sketch: exactly tqo_decode_attn, except that the value of token j is the JL
 * reconstruction above:  o' = sum_j p_j nv_j ( lut_V[codeV_j] + sqrt(pi/2)/m * gv_j * S^T sigmaV_j ).            */
void tqo_decode_attn_vq(int B, int H, int d, int m, int T_stride, double base, int layout, const float *q,
                        const int32_t *q_pos, const int32_t *seq_len, const float *pi_k, const float *pi_v,
                        const float *lut_k, const float *lut_v, const float *S, const uint8_t *k_codes,
                        const uint8_t *k_signs, const uint16_t *k_norm, const uint16_t *k_rnorm,
                        const uint8_t *v_codes, const uint16_t *v_norm, const uint8_t *v_signs,
                        const uint16_t *v_rnorm, double *out) {
  const int cb = 3 * d / 8, sb = m / 8;
  const double cq = sqrt(TQO_PI / 2.0) / (double)m;
#pragma omp parallel for schedule(dynamic)
  for (int unit = 0; unit < B * H; ++unit) {
    int b = unit / H, h = unit % H;
    int T = seq_len[b];
    double qv[256], qr[256], q2[256], z[256], o[256], sig[256], st[256];
    for (int i = 0; i < d; ++i) qv[i] = (double)q[(size_t)unit * d + i];
    tqo_rope(qv, d, (double)q_pos[b], base, layout, qr);
    matvec_f32(pi_k + (size_t)h * d * d, d, d, qr, q2);
    matvec_f32(S, m, d, q2, z);
    const float *luk = lut_k + (size_t)h * 8, *luv = lut_v + (size_t)h * 8;
    double *s = (double *)malloc(sizeof(double) * (size_t)(T > 0 ? T : 1));
    uint8_t codes[256], bits[256];
    double smax = -INFINITY;
    for (int j = 0; j < T; ++j) {
      size_t e = (size_t)unit * T_stride + j;
      tqo_unpack_codes(k_codes + e * cb, d, codes);
      tqo_unpack_bits(k_signs + e * sb, m, bits);
      double a = 0.0, bq = 0.0;
      for (int i = 0; i < d; ++i) a += q2[i] * (double)luk[codes[i]];
      for (int i = 0; i < m; ++i) bq += z[i] * (bits[i] ? 1.0 : -1.0);
      double n = tqo_f16_to_f64(k_norm[e]), g = tqo_f16_to_f64(k_rnorm[e]);
      s[j] = n * (a + cq * g * bq) / sqrt((double)d);
      if (s[j] > smax) smax = s[j];
    }
    double l = 0.0;
    for (int i = 0; i < d; ++i) o[i] = 0.0;
    for (int j = 0; j < T; ++j) {
      size_t e = (size_t)unit * T_stride + j;
      double p = exp(s[j] - smax);
      l += p;
      tqo_unpack_codes(v_codes + e * cb, d, codes);
      tqo_unpack_bits(v_signs + e * sb, m, bits);
      for (int i = 0; i < m; ++i) sig[i] = bits[i] ? 1.0 : -1.0;
      matvec_t_f32(S, m, d, sig, st); /* S^T sigma */
      double nv = tqo_f16_to_f64(v_norm[e]), gv = tqo_f16_to_f64(v_rnorm[e]);
      for (int i = 0; i < d; ++i) o[i] += p * nv * ((double)luv[codes[i]] + cq * gv * st[i]);
    }
    for (int i = 0; i < d; ++i) o[i] = T > 0 ? o[i] / l : 0.0;
    matvec_t_f32(pi_v + (size_t)h * d * d, d, d, o, out + (size_t)unit * d);
    free(s);
  }
}

/* Dequantise one cached vector back to the un-rotated space (the paper's two-step `fetch_unpacked`,
 * PAPER.md:120-122): x~ = n * PI^T ( lut[codes] ) — without the sketch term, which only exists as an
 * inner-product estimator.  Used by the brute-force attention pin.                                     */
void tqo_dequant_vector(const uint8_t *packed_codes, uint16_t norm_h, int d, const float *Pi, const float *lut8,
                        int unrotate, double *x_out) {
  uint8_t codes[256];
  double y[256];
  tqo_unpack_codes(packed_codes, d, codes);
  double n = tqo_f16_to_f64(norm_h);
  for (int i = 0; i < d; ++i) y[i] = n * (double)lut8[codes[i]];
  if (unrotate)
    matvec_t_f32(Pi, d, d, y, x_out);
  else
    memcpy(x_out, y, sizeof(double) * (size_t)d);
}

/* ---- exact attention on the original tensors (step 11; Eq. 1) -------------------------------------
 * out = softmax_j( <R_{p_q} q, R_j k_j> / sqrt(d) ) V, fp64.  k, v: [B][H][T_stride][d] fp32.           */
void tqo_dense_attn_ref(int B, int H, int d, int T_stride, double base, int layout, const float *q,
                        const int32_t *q_pos, const int32_t *seq_len, const float *k, const float *v,
                        double *out) {
#pragma omp parallel for schedule(dynamic)
  for (int unit = 0; unit < B * H; ++unit) {
    int b = unit / H;
    int T = seq_len[b];
    double qv[256], qr[256], kv[256], kr[256], o[256];
    for (int i = 0; i < d; ++i) qv[i] = (double)q[(size_t)unit * d + i];
    tqo_rope(qv, d, (double)q_pos[b], base, layout, qr);
    double *s = (double *)malloc(sizeof(double) * (size_t)(T > 0 ? T : 1));
    double smax = -INFINITY;
    for (int j = 0; j < T; ++j) {
      const float *kp = k + ((size_t)unit * T_stride + j) * d;
      for (int i = 0; i < d; ++i) kv[i] = (double)kp[i];
      tqo_rope(kv, d, (double)j, base, layout, kr);
      double a = 0.0;
      for (int i = 0; i < d; ++i) a += qr[i] * kr[i];
      s[j] = a / sqrt((double)d);
      if (s[j] > smax) smax = s[j];
    }
    double l = 0.0;
    for (int i = 0; i < d; ++i) o[i] = 0.0;
    for (int j = 0; j < T; ++j) {
      const float *vp = v + ((size_t)unit * T_stride + j) * d;
      double p = exp(s[j] - smax);
      l += p;
      for (int i = 0; i < d; ++i) o[i] += p * (double)vp[i];
    }
    for (int i = 0; i < d; ++i) out[(size_t)unit * d + i] = T > 0 ? o[i] / l : 0.0;
    free(s);
  }
}

/* ---- QJL inner-product estimator for one (q, r, S) (D2), exposed for the Monte-Carlo pin ----------
 * est = sqrt(pi/2)/m * |r| * < S q, sign(S r) >.                                                        */
double tqo_qjl_estimate(const double *q, const double *r, const float *S, int m, int d) {
  double z[256], sr[256], g2 = 0.0, acc = 0.0;
  matvec_f32(S, m, d, q, z);
  matvec_f32(S, m, d, r, sr);
  for (int i = 0; i < d; ++i) g2 += r[i] * r[i];
  for (int j = 0; j < m; ++j) acc += z[j] * (sr[j] >= 0.0 ? 1.0 : -1.0);
  return sqrt(TQO_PI / 2.0) / (double)m * sqrt(g2) * acc;
}

/* ---- Lloyd-Max for a zero-mean Gaussian (Eq. 5; configs[0] "Lloyd-Max on N(0,1/64)")
 * Alternate the two optimality conditions: t_k = (c_k + c_{k+1})/2 and c_k = E[x | t_{k-1} < x <= t_k]
 * with the closed-form truncated-Gaussian mean
 *   E[x | a < x <= b] = sigma * (phi(a/sigma) - phi(b/sigma)) / (Phi(b/sigma) - Phi(a/sigma)).
 * centroids[levels] ascending, thresholds[levels-1].  Returns the MSE  E[(x - c_bin(x))^2] / sigma^2.   */
static double npdf(double x) { return exp(-0.5 * x * x) / sqrt(2.0 * TQO_PI); }
static double ncdf(double x) { return 0.5 * erfc(-x / sqrt(2.0)); }

double tqo_lloyd_max_gauss(double sigma, int levels, int iters, double *centroids, double *thresholds) {
  double c[64], t[65];
  for (int k = 0; k < levels; ++k) c[k] = -2.0 + 4.0 * ((double)k + 0.5) / (double)levels; /* unit sigma */
  for (int it = 0; it < iters; ++it) {
    t[0] = -INFINITY;
    t[levels] = INFINITY;
    for (int k = 1; k < levels; ++k) t[k] = 0.5 * (c[k - 1] + c[k]);
    for (int k = 0; k < levels; ++k) {
      double a = t[k], b = t[k + 1];
      double pa = isinf(a) ? 0.0 : npdf(a), pb = isinf(b) ? 0.0 : npdf(b);
      double Pa = isinf(a) ? 0.0 : ncdf(a), Pb = isinf(b) ? 1.0 : ncdf(b);
      c[k] = (pa - pb) / (Pb - Pa);
    }
  }
  t[0] = -INFINITY;
  t[levels] = INFINITY;
  for (int k = 1; k < levels; ++k) t[k] = 0.5 * (c[k - 1] + c[k]);
  /* MSE = 1 - sum_k c_k^2 P_k  at a centroid fixed point (unit variance) */
  double mse = 1.0;
  for (int k = 0; k < levels; ++k) {
    double Pa = isinf(t[k]) ? 0.0 : ncdf(t[k]), Pb = isinf(t[k + 1]) ? 1.0 : ncdf(t[k + 1]);
    mse -= c[k] * c[k] * (Pb - Pa);
  }
  for (int k = 0; k < levels; ++k) centroids[k] = sigma * c[k];
  for (int k = 1; k < levels; ++k) thresholds[k - 1] = sigma * t[k];
  return mse;
}

/* ---- Lloyd-Max on samples = 1-D k-means ("SVD + K-means"; Eq. 5) ----------------------
 * samples must be sorted ascending.  Initialised at equally spaced quantiles.  Returns the mean squared
 * error.                                                                                               */
double tqo_lloyd_max_samples(const double *sorted, long n, int levels, int iters, double *centroids) {
  double c[64];
  for (int k = 0; k < levels; ++k) c[k] = sorted[(long)(((double)k + 0.5) / (double)levels * (double)n)];
  for (int it = 0; it < iters; ++it) {
    double sum[64];
    long cnt[64];
    for (int k = 0; k < levels; ++k) sum[k] = 0.0, cnt[k] = 0;
    int k = 0;
    for (long i = 0; i < n; ++i) {
      while (k < levels - 1 && sorted[i] > 0.5 * (c[k] + c[k + 1])) ++k;
      sum[k] += sorted[i];
      cnt[k] += 1;
    }
    for (k = 0; k < levels; ++k)
      if (cnt[k] > 0) c[k] = sum[k] / (double)cnt[k];
  }
  double mse = 0.0;
  int k = 0;
  for (long i = 0; i < n; ++i) {
    while (k < levels - 1 && sorted[i] > 0.5 * (c[k] + c[k + 1])) ++k;
    mse += (sorted[i] - c[k]) * (sorted[i] - c[k]);
  }
  for (k = 0; k < levels; ++k) centroids[k] = c[k];
  return mse / (double)n;
}
