// tq_calibrate_host.cpp — host-side calibration (not hot): head-wise SVD rotation,
// Lloyd-Max 8-point LUTs (Eq. 5), seeded Gaussian sketch S and the RoPE cos/sin table
// (BASELINE.json:north_star "host-side calibration").  Plain C++17, fp64 internally; shares no code with
// oracle/.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#include "../../include/tq.h"

namespace {

struct Rng {  // splitmix64 + Box-Muller: a counter-free seeded N(0,1) stream
  uint64_t s;
  explicit Rng(uint64_t seed) : s(seed) {}
  uint64_t next() {
    uint64_t z = (s += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
  }
  double uniform() { return ((next() >> 11) + 0.5) * (1.0 / 9007199254740992.0); }  // (0,1)
  double normal() {
    double u1 = uniform(), u2 = uniform();
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586476925 * u2);
  }
};

// Householder QR of a (d x d, row-major); returns Q with columns sign-fixed so that diag(R) > 0.
void qr_q(std::vector<double>& a, int d, std::vector<double>& q) {
  std::vector<double> vs((size_t)d * d, 0.0);  // Householder vectors, column j in vs[j*d ..]
  std::vector<double> rdiag(d, 0.0);
  for (int j = 0; j < d; ++j) {
    double nrm = 0.0;
    for (int i = j; i < d; ++i) nrm += a[(size_t)i * d + j] * a[(size_t)i * d + j];
    nrm = std::sqrt(nrm);
    double alpha = a[(size_t)j * d + j] > 0 ? -nrm : nrm;
    double* v = &vs[(size_t)j * d];
    for (int i = j; i < d; ++i) v[i] = a[(size_t)i * d + j];
    v[j] -= alpha;
    double vn = 0.0;
    for (int i = j; i < d; ++i) vn += v[i] * v[i];
    if (vn > 0) {
      for (int c = j; c < d; ++c) {
        double dot = 0.0;
        for (int i = j; i < d; ++i) dot += v[i] * a[(size_t)i * d + c];
        double f = 2.0 * dot / vn;
        for (int i = j; i < d; ++i) a[(size_t)i * d + c] -= f * v[i];
      }
    }
    rdiag[j] = a[(size_t)j * d + j];
  }
  // Q = H_0 H_1 ... H_{d-1} applied to I
  q.assign((size_t)d * d, 0.0);
  for (int i = 0; i < d; ++i) q[(size_t)i * d + i] = 1.0;
  for (int j = d - 1; j >= 0; --j) {
    const double* v = &vs[(size_t)j * d];
    double vn = 0.0;
    for (int i = j; i < d; ++i) vn += v[i] * v[i];
    if (vn == 0) continue;
    for (int c = 0; c < d; ++c) {
      double dot = 0.0;
      for (int i = j; i < d; ++i) dot += v[i] * q[(size_t)i * d + c];
      double f = 2.0 * dot / vn;
      for (int i = j; i < d; ++i) q[(size_t)i * d + c] -= f * v[i];
    }
  }
  for (int c = 0; c < d; ++c)
    if (rdiag[c] < 0)
      for (int i = 0; i < d; ++i) q[(size_t)i * d + c] = -q[(size_t)i * d + c];
}

// Cyclic Jacobi eigen-decomposition of a symmetric d x d matrix; eigenvectors in the columns of v.
void jacobi_eig(std::vector<double>& a, int d, std::vector<double>& v, std::vector<double>& w) {
  v.assign((size_t)d * d, 0.0);
  for (int i = 0; i < d; ++i) v[(size_t)i * d + i] = 1.0;
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int i = 0; i < d; ++i)
      for (int j = 0; j < d; ++j) (i == j ? diag : off) += a[(size_t)i * d + j] * a[(size_t)i * d + j];
    if (off <= 1e-30 * diag) break;
    for (int p = 0; p < d - 1; ++p)
      for (int q = p + 1; q < d; ++q) {
        double apq = a[(size_t)p * d + q];
        if (apq == 0.0) continue;
        double theta = (a[(size_t)q * d + q] - a[(size_t)p * d + p]) / (2.0 * apq);
        double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
        for (int k = 0; k < d; ++k) {
          double akp = a[(size_t)k * d + p], akq = a[(size_t)k * d + q];
          a[(size_t)k * d + p] = c * akp - s * akq;
          a[(size_t)k * d + q] = s * akp + c * akq;
        }
        for (int k = 0; k < d; ++k) {
          double apk = a[(size_t)p * d + k], aqk = a[(size_t)q * d + k];
          a[(size_t)p * d + k] = c * apk - s * aqk;
          a[(size_t)q * d + k] = s * apk + c * aqk;
        }
        for (int k = 0; k < d; ++k) {
          double vkp = v[(size_t)k * d + p], vkq = v[(size_t)k * d + q];
          v[(size_t)k * d + p] = c * vkp - s * vkq;
          v[(size_t)k * d + q] = s * vkp + c * vkq;
        }
      }
  }
  w.resize(d);
  for (int i = 0; i < d; ++i) w[i] = a[(size_t)i * d + i];
}

// PI = V^T of X = U Sigma V^T: rows of PI are the eigenvectors of X^T X by descending eigenvalue.
void svd_rotation(const float* X, int64_t n, int d, float* pi_out) {
  std::vector<double> g((size_t)d * d, 0.0);
  for (int64_t r = 0; r < n; ++r) {
    const float* x = X + r * d;
    for (int i = 0; i < d; ++i)
      for (int j = i; j < d; ++j) g[(size_t)i * d + j] += (double)x[i] * (double)x[j];
  }
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < i; ++j) g[(size_t)i * d + j] = g[(size_t)j * d + i];
  std::vector<double> v, w;
  jacobi_eig(g, d, v, w);
  std::vector<int> order(d);
  for (int i = 0; i < d; ++i) order[i] = i;
  std::sort(order.begin(), order.end(), [&](int a, int b) { return w[a] > w[b]; });
  for (int r = 0; r < d; ++r) {
    int c = order[r];
    // sign convention: largest-magnitude component positive (singular-vector signs are not unique)
    int arg = 0;
    for (int k = 1; k < d; ++k)
      if (std::fabs(v[(size_t)k * d + c]) > std::fabs(v[(size_t)arg * d + c])) arg = k;
    double sgn = v[(size_t)arg * d + c] < 0 ? -1.0 : 1.0;
    for (int k = 0; k < d; ++k) pi_out[(size_t)r * d + k] = (float)(sgn * v[(size_t)k * d + c]);
  }
}

double phi(double x) { return std::exp(-0.5 * x * x) * 0.3989422804014326779; }
double Phi(double x) { return 0.5 * std::erfc(-x * 0.7071067811865475244); }

// Lloyd-Max fixed point for N(0, sigma^2), 8 levels (Eq. 5): alternate midpoints / conditional means.
// Centroids are rounded to the nearest binary16-representable value (reading D15): the
// fused decode kernel then dequantises with exact fp16 tables (one 32-bit shared-memory read per code pair).  The
// change is 2^-12 relative, far below the quantiser's own error; every kernel also accepts LUTs that are not
// representable (two-term tables), so this is a calibration choice, not a format restriction.
float round_to_binary16(double x) {
  if (x == 0.0 || !std::isfinite(x)) return (float)x;
  int e;
  const double m = std::frexp(std::fabs(x), &e);  // |x| = m 2^e, m in [0.5, 1)
  if (e > 16) return (float)(x < 0 ? -65504.0 : 65504.0);
  const int qe = (e < -13 ? -24 : e - 11);        // spacing 2^qe: 11 significant bits, subnormals below 2^-14
  const double q = std::ldexp(std::nearbyint(std::ldexp(std::fabs(x), -qe)), qe);
  (void)m;
  return (float)(x < 0 ? -q : q);
}

void lloyd_max_gauss8(double sigma, float* lut8) {
  double c[8], t[9];
  for (int k = 0; k < 8; ++k) c[k] = -2.1 + 0.6 * k;
  for (int it = 0; it < 2000; ++it) {
    for (int k = 1; k < 8; ++k) t[k] = 0.5 * (c[k - 1] + c[k]);
    double delta = 0.0;
    for (int k = 0; k < 8; ++k) {
      double pa = k == 0 ? 0.0 : phi(t[k]), pb = k == 7 ? 0.0 : phi(t[k + 1]);
      double Pa = k == 0 ? 0.0 : Phi(t[k]), Pb = k == 7 ? 1.0 : Phi(t[k + 1]);
      double nc = (pa - pb) / (Pb - Pa);
      delta = std::max(delta, std::fabs(nc - c[k]));
      c[k] = nc;
    }
    if (delta < 1e-15) break;
  }
  for (int k = 0; k < 8; ++k) lut8[k] = round_to_binary16(sigma * c[k]);
}

// Lloyd-Max on samples (1-D k-means), samples sorted ascending.
void lloyd_max_samples8(std::vector<double>& s, float* lut8) {
  std::sort(s.begin(), s.end());
  const size_t n = s.size();
  double c[8];
  for (int k = 0; k < 8; ++k) c[k] = s[(size_t)((k + 0.5) / 8.0 * (double)n)];
  for (int it = 0; it < 200; ++it) {
    double sum[8] = {0}, cnt[8] = {0};
    int k = 0;
    for (size_t i = 0; i < n; ++i) {
      while (k < 7 && s[i] > 0.5 * (c[k] + c[k + 1])) ++k;
      sum[k] += s[i];
      cnt[k] += 1.0;
    }
    double delta = 0.0;
    for (k = 0; k < 8; ++k)
      if (cnt[k] > 0) {
        double nc = sum[k] / cnt[k];
        delta = std::max(delta, std::fabs(nc - c[k]));
        c[k] = nc;
      }
    if (delta < 1e-12) break;
  }
  for (int k = 0; k < 8; ++k) lut8[k] = round_to_binary16(c[k]);
}

void pooled_unit_coords(const float* X, int64_t n, int d, const float* pi, std::vector<double>& pool) {
  pool.clear();
  pool.reserve((size_t)n * d);
  std::vector<double> y(d);
  for (int64_t r = 0; r < n; ++r) {
    const float* x = X + r * d;
    double n2 = 0.0;
    for (int i = 0; i < d; ++i) {
      double acc = 0.0;
      for (int k = 0; k < d; ++k) acc += (double)pi[(size_t)i * d + k] * (double)x[k];
      y[i] = acc;
      n2 += acc * acc;
    }
    double nrm = std::sqrt(n2);
    if (nrm == 0) continue;
    for (int i = 0; i < d; ++i) pool.push_back(y[i] / nrm);
  }
}

// raw rotated coordinates y = PI x of every sample (paper-literal mode: the LUT lives on the activation scale)
void pooled_raw_coords(const float* X, int64_t n, int d, const float* pi, std::vector<double>& pool) {
  pool.clear();
  pool.reserve((size_t)n * d);
  for (int64_t r = 0; r < n; ++r) {
    const float* x = X + r * d;
    for (int i = 0; i < d; ++i) {
      double acc = 0.0;
      for (int k = 0; k < d; ++k) acc += (double)pi[(size_t)i * d + k] * (double)x[k];
      pool.push_back(acc);
    }
  }
}

int code_of(double u, const float* lut8) {
  int c = 0;
  for (int k = 0; k < 7; ++k) c += u > (double)(0.5f * (lut8[k] + lut8[k + 1])) ? 1 : 0;
  return c;
}

// e-bar of Eq. 7 [PAPER.md:176-179]: mean |y - lut[code(y)]| over the samples
double mean_abs_residual(const std::vector<double>& pool, const float* lut8) {
  double acc = 0.0;
  for (double y : pool) acc += std::fabs(y - (double)lut8[code_of(y, lut8)]);
  return pool.empty() ? 0.0 : acc / (double)pool.size();
}

// the same for y ~ N(0, sigma^2): sum over the cells [a, b] around centroid c of  int |y - c| dN, with
// int_p^q (y - c) dN = sigma (phi(p/sigma) - phi(q/sigma)) - c (Phi(q/sigma) - Phi(p/sigma))
double mean_abs_residual_gauss(double sigma, const float* lut8) {
  auto part = [&](double p, double q, double c) {  // p, q in units of sigma (may be +-inf)
    const double pp = std::isinf(p) ? 0.0 : phi(p), pq = std::isinf(q) ? 0.0 : phi(q);
    const double Pp = std::isinf(p) ? (p < 0 ? 0.0 : 1.0) : Phi(p), Pq = std::isinf(q) ? (q < 0 ? 0.0 : 1.0) : Phi(q);
    return sigma * (pp - pq) - c * (Pq - Pp);
  };
  double acc = 0.0;
  for (int k = 0; k < 8; ++k) {
    const double c = lut8[k];
    const double a = k == 0 ? -INFINITY : (double)(0.5f * (lut8[k - 1] + lut8[k])) / sigma;
    const double b = k == 7 ? INFINITY : (double)(0.5f * (lut8[k] + lut8[k + 1])) / sigma;
    const double cs = std::min(std::max(c / sigma, a), b);
    acc += -part(a, cs, c) + part(cs, b, c);
  }
  return acc;
}

void set_identity(float* M, int d) {
  for (int i = 0; i < d; ++i)
    for (int k = 0; k < d; ++k) M[(size_t)i * d + k] = i == k ? 1.f : 0.f;
}

}  // namespace

extern "C" int tq_calibrate_host(const tq_shape* shape, int32_t mode, const float* k_samples, const float* v_samples,
                                 int64_t n_samples, uint64_t seed, tq_params* out) {
  if (!shape || !out) return TQ_ERR_INVALID_ARG;
  const int L = shape->n_layers, H = shape->n_heads, d = shape->head_dim, m = shape->qjl_dim;
  if (L <= 0 || H <= 0 || shape->max_seq <= 0 || !(shape->rope_base > 0.f)) return TQ_ERR_INVALID_ARG;
  if ((d != 64 && d != 128) || m != d) return TQ_ERR_UNSUPPORTED;
  if (!out->pi_k || !out->pi_v || !out->lut_k || !out->lut_v || !out->S || !out->rope_cs) return TQ_ERR_INVALID_ARG;
  if (mode != 0 && mode != 1) return TQ_ERR_INVALID_ARG;
  if (mode == 0 && (!k_samples || !v_samples || n_samples < d)) return TQ_ERR_INVALID_ARG;
  const bool literal = shape->residual_mode == 1;  // the paper's Eq. 6-7 as printed (include/tq.h "Paper-literal mode")
  if (shape->residual_mode != 0 && shape->residual_mode != 1) return TQ_ERR_INVALID_ARG;
  if (literal && !out->ebar_k) return TQ_ERR_INVALID_ARG;

  Rng rs(seed ^ 0x5151515151515151ull);
  for (size_t i = 0; i < (size_t)m * d; ++i) out->S[i] = (float)rs.normal();
  if (literal) set_identity(out->S, d);  // Eq. 6: the sign of every residual coordinate

  for (int p = 0; p < shape->max_seq; ++p)
    for (int g = 0; g < d / 2; ++g) {
      double theta = std::pow((double)shape->rope_base, -2.0 * (double)g / (double)d);
      out->rope_cs[((size_t)p * (d / 2) + g) * 2 + 0] = (float)std::cos((double)p * theta);
      out->rope_cs[((size_t)p * (d / 2) + g) * 2 + 1] = (float)std::sin((double)p * theta);
    }

  if (mode == 1) {
    float lut[8];
    lloyd_max_gauss8(1.0 / std::sqrt((double)d), lut);
    Rng rk(seed ^ 0xA5A5A5A5A5A5A5A5ull), rv(seed ^ 0x3C3C3C3C3C3C3C3Cull);
    std::vector<double> g((size_t)d * d), q;
    for (int lh = 0; lh < L * H; ++lh) {
      for (auto& x : g) x = rk.normal();
      qr_q(g, d, q);
      for (size_t i = 0; i < (size_t)d * d; ++i) out->pi_k[(size_t)lh * d * d + i] = (float)q[i];
      for (auto& x : g) x = rv.normal();
      qr_q(g, d, q);
      for (size_t i = 0; i < (size_t)d * d; ++i) out->pi_v[(size_t)lh * d * d + i] = (float)q[i];
      for (int k = 0; k < 8; ++k) out->lut_k[(size_t)lh * 8 + k] = out->lut_v[(size_t)lh * 8 + k] = lut[k];
      if (literal) {
        set_identity(out->pi_v + (size_t)lh * d * d, d);  // values are not rotated
        out->ebar_k[lh] = (float)mean_abs_residual_gauss(1.0 / std::sqrt((double)d), lut);
      }
    }
    return TQ_OK;
  }
  std::vector<double> pool;
  for (int lh = 0; lh < L * H; ++lh) {
    const float* xk = k_samples + (size_t)lh * n_samples * d;
    const float* xv = v_samples + (size_t)lh * n_samples * d;
    float* pk = out->pi_k + (size_t)lh * d * d;
    float* pv = out->pi_v + (size_t)lh * d * d;
    svd_rotation(xk, n_samples, d, pk);
    if (literal) {  // LUTs on the raw (rotated) activations, values unrotated, e-bar over the key samples
      set_identity(pv, d);
      pooled_raw_coords(xk, n_samples, d, pk, pool);
      lloyd_max_samples8(pool, out->lut_k + (size_t)lh * 8);
      out->ebar_k[lh] = (float)mean_abs_residual(pool, out->lut_k + (size_t)lh * 8);
      pooled_raw_coords(xv, n_samples, d, pv, pool);
      lloyd_max_samples8(pool, out->lut_v + (size_t)lh * 8);
      continue;
    }
    svd_rotation(xv, n_samples, d, pv);
    pooled_unit_coords(xk, n_samples, d, pk, pool);
    if (pool.size() < 8) return TQ_ERR_INVALID_ARG;
    lloyd_max_samples8(pool, out->lut_k + (size_t)lh * 8);
    pooled_unit_coords(xv, n_samples, d, pv, pool);
    if (pool.size() < 8) return TQ_ERR_INVALID_ARG;
    lloyd_max_samples8(pool, out->lut_v + (size_t)lh * 8);
  }
  return TQ_OK;
}
