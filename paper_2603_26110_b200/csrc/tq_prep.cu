// tq_prep.cu — the small per-(batch, head) kernel in front of the streaming decode kernel.
//
// One CTA per (layer-in-call, batch, head) does, depending on the template flags,
//   kAppend : quantize-and-pack ONE new token (PAPER.md:111-116 per vector; BASELINE.json:configs[2]):
//             RoPE(k) -> PI_K -> norm, codes, residual -> S r -> bits;  PI_V v -> norm, codes; the words are
//             written into the tile slot seq_len[layer][b] and the last head of the batch entry bumps seq_len;
//   kQuery  : query preparation for the fused decode kernel (Eq. 4 moves PI to the query; north_star):
//             q'' = PI_K RoPE(q), z = S q''  -> workspace.
// tq_append = <true,false>, tq_decode_attn = <false,true>, tq_decode_step = <true,true>; in the fused form the
// rows of PI_K and S are fetched once and used for both the key and the query.
//
// These are latency-bound 3-stage chains (load -> mat-vec -> mat-vec); every matrix row a warp needs is
// requested before the first barrier so that the L2 latency is paid once, not once per stage.
#include "tq_common.cuh"

namespace tq {

__device__ __forceinline__ int code_of7(float u, const float* lut) {
  int c = 0;
#pragma unroll
  for (int q = 0; q < 7; ++q) c += (u > 0.5f * (lut[q] + lut[q + 1])) ? 1 : 0;
  return c;
}

// rows [8 warp, 8 warp + 8) of a row-major D x D matrix, lane holds elements lane + 32 j of each row
template <int D>
struct RowRegs {
  float m[8][D / 32];
  __device__ __forceinline__ void load(const float* __restrict__ M, int warp, int lane) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int j = 0; j < D / 32; ++j) m[r][j] = __ldg(M + (size_t)(warp * 8 + r) * D + lane + 32 * j);
  }
  // y[8 warp + r] = <row r, x>
  __device__ __forceinline__ void apply(const float* xsm, float* ysm, int warp, int lane) const {
    float xr[D / 32];
#pragma unroll
    for (int j = 0; j < D / 32; ++j) xr[j] = xsm[lane + 32 * j];
    float p[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      p[r] = 0.f;
#pragma unroll
      for (int j = 0; j < D / 32; ++j) p[r] = fmaf(m[r][j], xr[j], p[r]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int r = 0; r < 8; ++r) p[r] += __shfl_xor_sync(0xffffffffu, p[r], o);
    if (lane == 0) {
#pragma unroll
      for (int r = 0; r < 8; ++r) ysm[warp * 8 + r] = p[r];
    }
  }
};

struct PrepArgs {
  CacheView cv;
  const float *pi_k, *pi_v, *lut_k, *lut_v, *S, *rope_cs;  // full [L][H]... arrays
  const void *q, *k, *v;                                    // [Lc][B][H][D] each (k, v: append; q: query)
  void* out;                                                // [Lc][B][H][D] (zeroed here for empty caches)
  const int32_t* q_pos;                                     // [Lc][B] or nullptr
  float* qrot;                                              // workspace [units][2 D]
  int layer_begin, rope_layout;
};

template <int D, typename T, bool kAppend, bool kQuery>
__global__ void __launch_bounds__(4 * D) prep_kernel(PrepArgs a) {
  using Lo = Layout<D>;
  constexpr int NT = 4 * D;  // 8 rows per warp
  constexpr int HP = D / 2;
  constexpr float kInvSqrtD = D == 64 ? 0.125f : 0.08838834764831845f;
  constexpr float kScaleK = 1.4426950408889634f * kInvSqrtD;             // log2(e) / sqrt(d)
  constexpr float kScaleS = kScaleK * 1.2533141373155003f / (float)D;  // ... * sqrt(pi/2) / m, m = D
  __shared__ float xk[D], xq[D], xv[D], yk[D], yq[D], yv[D], r[D], sr[D], zq[D];
  __shared__ unsigned char cK[D], cV[D], bK[D];
  __shared__ float nrm[4];
  __shared__ float lutK[8], lutV[8];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int uc = blockIdx.x;
  const int B = a.cv.B, H = a.cv.H;
  const int lc = uc / (B * H), bh = uc % (B * H), b = bh / H, h = bh % H;
  const int layer = a.layer_begin + lc;
  const int lb = layer * B + b;
  const int len0 = a.cv.seq_len[lb];
  const bool full = kAppend && len0 >= a.cv.max_seq;
  const int len1 = (kAppend && !full) ? len0 + 1 : len0;  // length the decode kernel will see
  // RoPE positions: the appended key sits at index len0; the query defaults to the newest cached token
  int qpos = a.q_pos ? a.q_pos[lc * B + b] : len1 - 1;
  qpos = max(0, min(qpos, a.cv.max_seq - 1));
  const int kpos = min(len0, a.cv.max_seq - 1);

  // ---- every global load that does not depend on a result, up front
  RowRegs<D> Mk, Mv, Ms;
  const size_t lh = (size_t)layer * H + h;
  Mk.load(a.pi_k + lh * D * D, warp, lane);
  if (kAppend) Mv.load(a.pi_v + lh * D * D, warp, lane);
  Ms.load(a.S, warp, lane);
  if (tid < 8) lutK[tid] = a.lut_k[lh * 8 + tid];
  if (tid >= 32 && tid < 40) lutV[tid - 32] = a.lut_v[lh * 8 + tid - 32];
  if (tid < HP) {
    const int g = tid;
    const int ia = a.rope_layout == 0 ? 2 * g : g, ib = a.rope_layout == 0 ? 2 * g + 1 : g + HP;
    if (kAppend) {
      const T* kp = reinterpret_cast<const T*>(a.k) + (size_t)uc * D;
      const float xa = load_as_float<T>(kp + ia), xb = load_as_float<T>(kp + ib);
      const float2 cs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)kpos * HP + g) * 2);
      xk[ia] = xa * cs.x - xb * cs.y;
      xk[ib] = xa * cs.y + xb * cs.x;
    }
    if (kQuery) {
      const T* qp = reinterpret_cast<const T*>(a.q) + (size_t)uc * D;
      const float xa = load_as_float<T>(qp + ia), xb = load_as_float<T>(qp + ib);
      const float2 cs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)qpos * HP + g) * 2);
      xq[ia] = xa * cs.x - xb * cs.y;
      xq[ib] = xa * cs.y + xb * cs.x;
    }
  } else if (kAppend && tid >= NT / 2 && tid < NT / 2 + D) {
    xv[tid - NT / 2] = load_as_float<T>(reinterpret_cast<const T*>(a.v) + (size_t)uc * D + tid - NT / 2);
  }
  __syncthreads();

  // ---- stage 1: rotations
  if (kAppend) Mk.apply(xk, yk, warp, lane);
  if (kQuery) Mk.apply(xq, yq, warp, lane);
  if (kAppend) Mv.apply(xv, yv, warp, lane);
  __syncthreads();
  if (kQuery) {
    float* dst = a.qrot + (size_t)uc * 2 * D;
    if (tid < D) dst[tid] = yq[tid] * kScaleK;  // logits in log2 units
    if (len1 <= 0 && tid < D) {  // empty cache: no tile for this unit in the streaming kernel, out = 0
      T* outp = reinterpret_cast<T*>(a.out) + (size_t)uc * D;
      if constexpr (sizeof(T) == 2) outp[tid] = __float2half_rn(0.f);
      else outp[tid] = 0.f;
    }
  }
  if (kAppend) {
    if (warp < 2) {  // warp 0: |y_k|, warp 1: |y_v|
      const float* y = warp == 0 ? yk : yv;
      float p = 0.f;
#pragma unroll
      for (int i = lane; i < D; i += 32) p = fmaf(y[i], y[i], p);
      p = warp_sum(p);
      if (lane == 0) nrm[warp] = sqrtf(p);
    }
    __syncthreads();
    const float n = nrm[0], nv = nrm[1];
    if (tid < D) {
      const float u = n > 0.f ? yk[tid] / n : 0.f;
      const int c = code_of7(u, lutK);
      cK[tid] = (unsigned char)c;
      r[tid] = u - lutK[c];
    } else if (tid >= NT / 2 && tid < NT / 2 + D) {
      const int i = tid - NT / 2;
      const float u = nv > 0.f ? yv[i] / nv : 0.f;
      cV[i] = (unsigned char)code_of7(u, lutV);
    }
    __syncthreads();
    if (warp == 0) {
      float p = 0.f;
#pragma unroll
      for (int i = lane; i < D; i += 32) p = fmaf(r[i], r[i], p);
      p = warp_sum(p);
      if (lane == 0) nrm[2] = sqrtf(p);
    }
  }
  // ---- stage 2: sketch of the residual / of the rotated query
  if (kAppend) Ms.apply(r, sr, warp, lane);
  if (kQuery) Ms.apply(yq, zq, warp, lane);
  __syncthreads();
  if (kQuery && tid < D)  // log2(e)/sqrt(d) * sqrt(pi/2)/m, m = D
    a.qrot[(size_t)uc * 2 * D + D + tid] = zq[tid] * kScaleS;
  if (kAppend) {
    if (tid < D) bK[tid] = sr[tid] >= 0.f ? 1 : 0;
    __syncthreads();
    if (!full) {  // ---- assemble this token's words (device layout, include/tq.h)
      const int pos = len0;
      const size_t unit = (size_t)layer * B * H + bh;
      unsigned char* tp = a.cv.tiles + unit * a.cv.stream_bytes + (size_t)(pos / kTile) * Lo::kTileBytes;
      const int slot = pos % kTile;
      if (tid < Lo::KCW) {
        const int w = tid;
        unsigned long long word = 0;
        const int k_lo = (32 * w) / 6, k_hi = (32 * w + 31) / 6;
        for (int kf = k_lo; kf <= k_hi; ++kf) {
          const int g = (kf + slot) % Lo::P;
          unsigned long long f = cK[2 * g] | ((unsigned)cK[2 * g + 1] << 3);
          const int sh = 6 * kf - 32 * w;
          word |= sh >= 0 ? (f << sh) : (f >> (-sh));
        }
        *reinterpret_cast<unsigned*>(tp + Lo::kOffKC + word_offset(Lo::KCW, w, slot)) = (unsigned)word;
      } else if (tid >= 32 && tid < 32 + Lo::KSW) {
        const int w = tid - 32;
        unsigned word = 0;
        for (int kn = 0; kn < 8; ++kn) {
          const int ng = (8 * w + kn + slot) % Lo::NG;
          unsigned nib = bK[4 * ng] | (bK[4 * ng + 1] << 1) | (bK[4 * ng + 2] << 2) | (bK[4 * ng + 3] << 3);
          word |= nib << (4 * kn);
        }
        *reinterpret_cast<unsigned*>(tp + Lo::kOffKS + word_offset(Lo::KSW, w, slot)) = word;
      } else if (tid >= 64 && tid < 64 + Lo::P) {
        // V: pair group g lives in lane (g mod 32)'s string at bits [192 part + 6 slot, +6): read-modify-write
        const int g = tid - 64, vl = g % kTile, part = g / kTile;
        const unsigned f = cV[2 * g] | ((unsigned)cV[2 * g + 1] << 3);
        const int bit = 192 * part + 6 * slot, s = bit & 31;
        unsigned* p0 = reinterpret_cast<unsigned*>(tp + Lo::kOffVC + word_offset(Lo::KCW, bit >> 5, vl));
        *p0 = (*p0 & ~(63u << s)) | (f << s);
        if (s > 26) {
          unsigned* p1 = reinterpret_cast<unsigned*>(tp + Lo::kOffVC + word_offset(Lo::KCW, (bit >> 5) + 1, vl));
          *p1 = (*p1 & ~(63u >> (32 - s))) | (f >> (32 - s));
        }
      } else if (tid == 192) {
        reinterpret_cast<unsigned short*>(tp + Lo::kOffKN)[slot] = f32_to_f16_bits_clamped(nrm[0]);
        reinterpret_cast<unsigned short*>(tp + Lo::kOffKR)[slot] = f32_to_f16_bits_clamped(nrm[2]);
        reinterpret_cast<unsigned short*>(tp + Lo::kOffVN)[slot] = f32_to_f16_bits_clamped(nrm[1]);
      }
    }
    // ---- arrival: the last head of batch entry b publishes the new length
    __syncthreads();
    if (tid == 0) {
      __threadfence();
      const int old = atomicAdd(&a.cv.arrive[lb], 1);
      if (old == H - 1) {
        a.cv.arrive[lb] = 0;
        if (full) atomicExch(a.cv.status, (int)TQ_ERR_CAPACITY);
        else a.cv.seq_len[lb] = len0 + 1;
        __threadfence();
      }
    }
  }
}

template <int D, typename T>
static cudaError_t launch_prep_t(const PrepArgs& a, int units, bool do_append, bool do_query, cudaStream_t st) {
  if (do_append && do_query) prep_kernel<D, T, true, true><<<units, 4 * D, 0, st>>>(a);
  else if (do_append) prep_kernel<D, T, true, false><<<units, 4 * D, 0, st>>>(a);
  else prep_kernel<D, T, false, true><<<units, 4 * D, 0, st>>>(a);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_prep(const DecodeArgs& d, const void* k, const void* v, int D, bool do_append, bool do_query,
                        cudaStream_t st) {
  PrepArgs a;
  a.cv = d.cv;
  a.pi_k = d.pi_k;
  a.pi_v = d.pi_v;
  a.lut_k = d.lut_k;
  a.lut_v = d.lut_v;
  a.S = d.S;
  a.rope_cs = d.rope_cs;
  a.q = d.q;
  a.k = k;
  a.v = v;
  a.out = d.out;
  a.q_pos = d.q_pos;
  a.qrot = d.qrot;
  a.layer_begin = d.layer_begin;
  a.rope_layout = d.rope_layout;
  const int units = d.n_layers_call * d.cv.B * d.cv.H;
  if (D == 64)
    return d.dt == TQ_F16 ? launch_prep_t<64, __half>(a, units, do_append, do_query, st)
                          : launch_prep_t<64, float>(a, units, do_append, do_query, st);
  return d.dt == TQ_F16 ? launch_prep_t<128, __half>(a, units, do_append, do_query, st)
                        : launch_prep_t<128, float>(a, units, do_append, do_query, st);
}

}  // namespace tq
