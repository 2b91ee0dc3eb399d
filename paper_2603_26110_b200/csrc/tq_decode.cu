// tq_decode.cu — fused decode attention over the packed 3-bit cache (sm_100a, CUDA cores by design:
// a one-query GEMV over a packed stream is bound by HBM bandwidth and by instruction issue, not by
// tensor throughput — DESIGN.md "Decode kernel").
//
// Algorithm 1 of the paper re-associated as BASELINE.json:north_star asks: the query is
// rotated once (q'' = PI_K RoPE(q), z = S q''; Eq. 4 moves PI from every key to the query), then the cache
// is streamed exactly once:
//   logit_j = n_j ( <q'', lut_K[codes_j]> + sqrt(pi/2)/m * g_j * <z, sigma_j> ) / sqrt(d)
//   online softmax (running max m, sum l), o' += p_j * nv_j * lut_V[codesV_j];   out = PI_V^T (o' / l).
//
// Mapping: lane = token.  Each lane owns one token of a 32-token tile and walks its 6-bit code-pair fields.
//   * <q'', lut_K[.]> becomes P = d/2 table reads: Ktab[field][col] = q''_{2g} lut[c0] + q''_{2g+1} lut[c1],
//     col = (lane + k) so that the 32 lanes always hit 32 different banks (the cache stores field g at
//     position (g - lane) mod P for exactly this reason);
//   * <z, sigma> becomes d/4 reads of a 16-entry nibble table with the same rotation;
//   * V is dequantised two coordinates per 64-bit table read ([field][lane] float2, conflict free) and
//     accumulated into d fp32 registers per lane; lanes are summed once per warp at the end.
// Split-K over the sequence: grid = units x nsplit CTAs; the last CTA to finish a unit merges the partial
// (m, l, o') triples and applies PI_V^T.
#include <utility>

#include "tq_common.cuh"

namespace tq {


// ------------------------------------------------------------------------------------------ query prep
template <int D, typename T>
__global__ void __launch_bounds__(128) decode_prep_kernel(DecodeArgs a) {
  __shared__ float x[D], y[D];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int uc = blockIdx.x;
  const int BH = a.cv.B * a.cv.H;
  const int lc = uc / BH, bh = uc % BH, b = bh / a.cv.H, h = bh % a.cv.H;
  const int layer = a.layer_begin + lc;
  int pos = a.q_pos ? a.q_pos[lc * a.cv.B + b] : a.cv.seq_len[layer * a.cv.B + b] - 1;
  pos = max(0, min(pos, a.cv.max_seq - 1));
  constexpr int HP = D / 2;
  const T* qp = reinterpret_cast<const T*>(a.q) + (size_t)uc * D;
  for (int g = tid; g < HP; g += 128) {
    int ia = a.rope_layout == 0 ? 2 * g : g, ib = a.rope_layout == 0 ? 2 * g + 1 : g + HP;
    float xa = load_as_float<T>(qp + ia), xb = load_as_float<T>(qp + ib);
    float2 cs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)pos * HP + g) * 2);
    x[ia] = xa * cs.x - xb * cs.y;
    x[ib] = xa * cs.y + xb * cs.x;
  }
  __syncthreads();
  const float* Pk = a.pi_k + ((size_t)layer * a.cv.H + h) * D * D;
  for (int i = warp; i < D; i += 4) {
    float p = 0.f;
#pragma unroll
    for (int k = lane; k < D; k += 32) p = fmaf(Pk[(size_t)i * D + k], x[k], p);
    p = warp_sum(p);
    if (lane == 0) y[i] = p;
  }
  __syncthreads();
  float* dst = a.qrot + (size_t)uc * 2 * D;
  for (int i = tid; i < D; i += 128) dst[i] = y[i];
  for (int j = warp; j < D; j += 4) {
    float p = 0.f;
#pragma unroll
    for (int k = lane; k < D; k += 32) p = fmaf(a.S[(size_t)j * D + k], y[k], p);
    p = warp_sum(p);
    if (lane == 0) dst[D + j] = p;
  }
}

// ------------------------------------------------------------------------------------------ smem helpers
template <int IMM>
__device__ __forceinline__ float lds_f32(unsigned addr) {
  float v;
  asm("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(addr), "n"(IMM));
  return v;
}
__device__ __forceinline__ float2 lds_f32x2(unsigned addr) {
  float2 v;
  asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
  return v;
}

// bits [BIT, BIT+NB) of the little-endian word string w, moved to bit position LS and masked
template <int LS, int BIT, int NB, int NW>
__device__ __forceinline__ unsigned field_at(const unsigned (&w)[NW]) {
  constexpr int wi = BIT >> 5, s = BIT & 31;
  constexpr unsigned mask = ((1u << NB) - 1u) << LS;
  unsigned v;
  if constexpr (s + NB > 32)
    v = __funnelshift_r(w[wi], w[(wi + 1) % NW], s - LS);
  else if constexpr (s >= LS)
    v = w[wi] >> (s - LS);
  else
    v = w[wi] << (LS - s);
  return v & mask;
}

template <int D>
struct DecodeCfg {
  using Lo = Layout<D>;
  static constexpr int NCK = D == 64 ? 64 : 128;        // columns of the K table (>= P + 31)
  static constexpr int LSK = D == 64 ? 8 : 9;           // log2(NCK * 4)
  static constexpr int kKtabBytes = 64 * NCK * 4;        // 16 KB | 32 KB
  static constexpr int kVtabBytes = 64 * 32 * 8;         // 16 KB
  static constexpr int kStabBytes = 16 * 64 * 4;         // 4 KB
  static constexpr int kAlign = kKtabBytes;              // base alignment that makes the OR-addressing valid
  static constexpr int kRedFloats = 4 * (D + 2) + D + 4;  // per-warp (m, l, o'), merged o, flags
  static constexpr int kSmemBytes = kAlign + kKtabBytes + kVtabBytes + kStabBytes + kRedFloats * 4;
};

template <int D, int... K>
__device__ __forceinline__ float k_score(const unsigned (&kw)[Layout<D>::KCW], unsigned kbase,
                                         std::integer_sequence<int, K...>) {
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  ((acc[K & 3] += lds_f32<4 * K>(field_at<DecodeCfg<D>::LSK, 6 * K, 6>(kw) | kbase)), ...);
  return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}

template <int D, int... K>
__device__ __forceinline__ float s_score(const unsigned (&sw)[Layout<D>::KSW], unsigned sbase,
                                         std::integer_sequence<int, K...>) {
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  ((acc[K & 3] += lds_f32<4 * K>(field_at<8, 4 * K, 4>(sw) | sbase)), ...);
  return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}

template <int D, int... K>
__device__ __forceinline__ void v_accum(const unsigned (&vw)[Layout<D>::KCW], unsigned vbase, float w, float (&o)[D],
                                        std::integer_sequence<int, K...>) {
  (([&] {
     float2 lv = lds_f32x2(field_at<8, 6 * K, 6>(vw) | vbase);
     o[2 * K] = fmaf(w, lv.x, o[2 * K]);
     o[2 * K + 1] = fmaf(w, lv.y, o[2 * K + 1]);
   }()),
   ...);
}

// one token's packed words, as loaded by the lane that owns it
template <int D>
struct TokenWords {
  unsigned kw[Layout<D>::KCW];
  unsigned sw[Layout<D>::KSW];
  unsigned vw[Layout<D>::KCW];
  unsigned short kn, kr, vn;
};

template <int W>
__device__ __forceinline__ void load_words(unsigned (&dst)[W], const unsigned char* sec, int lane) {
#pragma unroll
  for (int c = 0; c < W / 4; ++c) {
    uint4 v = __ldg(reinterpret_cast<const uint4*>(sec + c * 16 * kTile + lane * 16));
    dst[4 * c] = v.x;
    dst[4 * c + 1] = v.y;
    dst[4 * c + 2] = v.z;
    dst[4 * c + 3] = v.w;
  }
  if constexpr (W % 4 == 2) {
    uint2 v = __ldg(reinterpret_cast<const uint2*>(sec + (W / 4) * 16 * kTile + lane * 8));
    dst[W - 2] = v.x;
    dst[W - 1] = v.y;
  }
}

template <int D>
__device__ __forceinline__ void load_token(TokenWords<D>& t, const unsigned char* tp, int lane) {
  using Lo = Layout<D>;
  load_words<Lo::KCW>(t.kw, tp + Lo::kOffKC, lane);
  load_words<Lo::KSW>(t.sw, tp + Lo::kOffKS, lane);
  load_words<Lo::KCW>(t.vw, tp + Lo::kOffVC, lane);
  t.kn = __ldg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffKN) + lane);
  t.kr = __ldg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffKR) + lane);
  t.vn = __ldg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffVN) + lane);
}

// Sum o[0..N) over the 32 lanes; afterwards lane holds elements [ (N/32) * lane, (N/32) * (lane+1) ) in o[0..N/32).
template <int N>
__device__ __forceinline__ void lanes_transpose_sum(float (&o)[N], int lane) {
  static_assert(N % 32 == 0, "");
#pragma unroll
  for (int stage = 0; stage < 5; ++stage) {
    const int off = 16 >> stage;
    const int half = N >> (stage + 1);  // elements kept after this stage
    const bool upper = (lane & off) != 0;
#pragma unroll
    for (int i = 0; i < N / 2; ++i) {
      if (i < half) {
        float send = upper ? o[i] : o[i + half];
        float keep = upper ? o[i + half] : o[i];
        o[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
      }
    }
  }
}

constexpr float kLazyThreshold = 16.0f;  // log2 units: rescale only when the running max grows by > 2^16

template <int D, typename TIO>
__global__ void __launch_bounds__(128) decode_main_kernel(DecodeArgs a) {
  using Lo = Layout<D>;
  using Cfg = DecodeCfg<D>;
  extern __shared__ unsigned char smem_raw[];
  const unsigned raw = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned ktab = (raw + Cfg::kAlign - 1) & ~(unsigned)(Cfg::kAlign - 1);
  const unsigned vtab = ktab + Cfg::kKtabBytes;
  const unsigned stab = vtab + Cfg::kVtabBytes;
  unsigned char* gen = smem_raw + (ktab - raw);  // generic pointer to the aligned region
  float* Ktab = reinterpret_cast<float*>(gen);
  float2* Vtab = reinterpret_cast<float2*>(gen + Cfg::kKtabBytes);
  float* Stab = reinterpret_cast<float*>(gen + Cfg::kKtabBytes + Cfg::kVtabBytes);
  float* red = reinterpret_cast<float*>(gen + Cfg::kKtabBytes + Cfg::kVtabBytes + Cfg::kStabBytes);
  float* omerged = red + 4 * (D + 2);  // [D] + flags
  int* flag = reinterpret_cast<int*>(omerged + D);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int uc = blockIdx.x / a.nsplit, split = blockIdx.x % a.nsplit;
  const int BH = a.cv.B * a.cv.H;
  const int lc = uc / BH, bh = uc % BH, b = bh / a.cv.H, h = bh % a.cv.H;
  const int layer = a.layer_begin + lc;
  const int T = a.cv.seq_len[layer * a.cv.B + b];
  const int ntiles = (T + kTile - 1) / kTile;
  const int tps = (ntiles + a.nsplit - 1) / a.nsplit;
  const int tile_begin = split * tps;
  const int tile_end = min(ntiles, tile_begin + tps);

  // ---- tables (pre-scaled so that the logit comes out in log2 units)
  {
    const float* qr = a.qrot + (size_t)uc * 2 * D;
    const float* lk = a.lut_k + ((size_t)layer * a.cv.H + h) * 8;
    const float* lv = a.lut_v + ((size_t)layer * a.cv.H + h) * 8;
    const float sc_k = 1.4426950408889634f * rsqrtf((float)D);
    const float sc_s = sc_k * 1.2533141373155003f / (float)D;  // sqrt(pi/2) / m, m = D
    for (int idx = tid; idx < 64 * Cfg::NCK; idx += 128) {
      const int e = idx / Cfg::NCK, c = idx % Cfg::NCK, g = c % Lo::P;
      Ktab[idx] = fmaf(qr[2 * g], lk[e & 7], qr[2 * g + 1] * lk[e >> 3]) * sc_k;
    }
    for (int idx = tid; idx < 16 * 64; idx += 128) {
      const int e = idx / 64, c = idx % 64, n = c % Lo::NG;
      float s = 0.f;
#pragma unroll
      for (int bb = 0; bb < 4; ++bb) s += ((e >> bb) & 1) ? qr[D + 4 * n + bb] : -qr[D + 4 * n + bb];
      Stab[idx] = s * sc_s;
    }
    for (int idx = tid; idx < 64 * 32; idx += 128) {
      const int e = idx / 32;
      Vtab[idx] = make_float2(lv[e & 7], lv[e >> 3]);
    }
  }
  __syncthreads();

  const unsigned kbase = ktab + lane * 4, sbase = stab + lane * 4, vbase = vtab + lane * 8;
  const size_t unit = (size_t)layer * BH + bh;
  const unsigned char* stream = a.cv.tiles + unit * a.cv.stream_bytes;

  float o[D];
#pragma unroll
  for (int i = 0; i < D; ++i) o[i] = 0.f;
  float m = -INFINITY, l = 0.f;

  TokenWords<D> cur, nxt;
  int tile = tile_begin + warp;
  if (tile < tile_end) load_token<D>(cur, stream + (size_t)tile * Lo::kTileBytes, lane);
  for (; tile < tile_end; tile += 4) {
    const bool has_next = tile + 4 < tile_end;
    if (has_next) load_token<D>(nxt, stream + (size_t)(tile + 4) * Lo::kTileBytes, lane);
    const bool valid = tile * kTile + lane < T;
    const float sa = k_score<D>(cur.kw, kbase, std::make_integer_sequence<int, Lo::P>{});
    const float sb = s_score<D>(cur.sw, sbase, std::make_integer_sequence<int, Lo::NG>{});
    float s2 = f16_bits_to_f32(cur.kn) * fmaf(f16_bits_to_f32(cur.kr), sb, sa);
    s2 = valid ? s2 : -INFINITY;
    const float tmax = warp_max(s2);  // finite: slot 0 of every processed tile is valid
    if (tmax > m + kLazyThreshold) {  // warp-uniform; also taken on the first tile (m = -inf)
      const float f = exp2f(m - tmax);  // 0 on the first tile
      l *= f;
#pragma unroll
      for (int i = 0; i < D; ++i) o[i] *= f;
      m = tmax;
    }
    const float p = exp2f(s2 - m);  // invalid lanes: exp2(-inf) = 0
    l += p;
    const float w = valid ? p * f16_bits_to_f32(cur.vn) : 0.f;
    v_accum<D>(cur.vw, vbase, w, o, std::make_integer_sequence<int, Lo::P>{});
    if (has_next) cur = nxt;
  }

  // ---- per-warp reduction over lanes, then over the CTA's warps
  lanes_transpose_sum<D>(o, lane);
  l = warp_sum(l);
  float* wr = red + warp * (D + 2);
  if (lane == 0) {
    wr[0] = m;
    wr[1] = l;
  }
#pragma unroll
  for (int i = 0; i < D / 32; ++i) wr[2 + (D / 32) * lane + i] = o[i];
  __syncthreads();
  float M = fmaxf(fmaxf(red[0], red[D + 2]), fmaxf(red[2 * (D + 2)], red[3 * (D + 2)]));
  float Lsum = 0.f, oi = 0.f;
  if (tid < D) {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const float mw = red[w * (D + 2)];
      const float f = mw == -INFINITY ? 0.f : exp2f(mw - M);
      Lsum = fmaf(red[w * (D + 2) + 1], f, Lsum);
      oi = fmaf(red[w * (D + 2) + 2 + tid], f, oi);
    }
  }
  TIO* outp = reinterpret_cast<TIO*>(a.out) + (size_t)uc * D;
  const float* Pv = a.pi_v + ((size_t)layer * a.cv.H + h) * D * D;
  if (a.nsplit > 1) {
    float* part = a.partials + ((size_t)uc * a.nsplit + split) * (D + 2);
    if (tid < D) part[2 + tid] = oi;
    if (tid == 0) {
      part[0] = M;
      part[1] = Lsum;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      int old = atomicAdd(&a.counters[uc], 1);
      *flag = (old == a.nsplit - 1);
      if (old == a.nsplit - 1) a.counters[uc] = 0;
    }
    __syncthreads();
    if (!*flag) return;
    __threadfence();
    const float* pp = a.partials + (size_t)uc * a.nsplit * (D + 2);
    M = -INFINITY;
    for (int s = 0; s < a.nsplit; ++s) M = fmaxf(M, __ldcg(pp + s * (D + 2)));
    Lsum = 0.f;
    oi = 0.f;
    if (tid < D) {
      for (int s = 0; s < a.nsplit; ++s) {
        const float ms = __ldcg(pp + s * (D + 2));
        const float f = ms == -INFINITY ? 0.f : exp2f(ms - M);
        Lsum = fmaf(__ldcg(pp + s * (D + 2) + 1), f, Lsum);
        oi = fmaf(__ldcg(pp + s * (D + 2) + 2 + tid), f, oi);
      }
    }
  }
  // ---- finalise: out = PI_V^T (o' / l); an empty cache gives 0
  if (tid < D) omerged[tid] = Lsum > 0.f ? oi / Lsum : 0.f;
  __syncthreads();
  if (tid < D) {
    float r = 0.f;
#pragma unroll 8
    for (int k = 0; k < D; ++k) r = fmaf(Pv[(size_t)k * D + tid], omerged[k], r);
    if constexpr (sizeof(TIO) == 2)
      outp[tid] = __float2half_rn(r);
    else
      outp[tid] = r;
  }
}

// ------------------------------------------------------------------------------------------ launchers
template <int D, typename T>
static cudaError_t launch_decode_t(const DecodeArgs& a, cudaStream_t st) {
  const int units = a.n_layers_call * a.cv.B * a.cv.H;
  decode_prep_kernel<D, T><<<units, 128, 0, st>>>(a);
  count_launch();
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  constexpr int smem = DecodeCfg<D>::kSmemBytes;
  e = cudaFuncSetAttribute(decode_main_kernel<D, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  decode_main_kernel<D, T><<<units * a.nsplit, 128, smem, st>>>(a);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_decode(const DecodeArgs& a, int D, cudaStream_t st) {
  if (D == 64)
    return a.dt == TQ_F16 ? launch_decode_t<64, __half>(a, st) : launch_decode_t<64, float>(a, st);
  return a.dt == TQ_F16 ? launch_decode_t<128, __half>(a, st) : launch_decode_t<128, float>(a, st);
}

}  // namespace tq
