// tq_quantize.cu — the fp32 CUDA-core quantize-and-pack kernel (prefill tiles), sm_100a.
//
// NOT the product kernel: tq_quantize_pack runs the tcgen05 kernel of tq_quantize_tc.cu, and the single-token append
// lives in tq_prep.cu.  This file is the independent second implementation the tests cross-check the tensor-core
// kernel against (test_tensor_core_quantize_agrees_with_cuda_core_kernel); it is reached only through the test knob
// tq_debug_set_quantize_impl(1), implements the default mode only (no paper-literal mode, no V-side sketch) and is
// never timed by bench.py.
//
// Per vector (PAPER.md:111-116 prefill steps 1,3,4; §3.3 Eq. 5; §3.4 Eq. 6 in the sign(S r) form of
// BASELINE.json:north_star): RoPE (keys) -> y = PI x' -> n = |y|, u = y / n -> code_i = #{k: u_i > t_k}
// -> r = u - lut[code], |r|, bits_j = [(S r)_j >= 0] -> device tile layout (include/tq.h).
//
// Prefill kernel: one CTA owns a run of 32-token tiles of one (batch, head).  PI_K, S and PI_V stay
// resident in shared memory (transposed, [k][i]) for the whole run; each tile is a
// (32 tokens x D) x (D x D) fp32 register-tiled GEMM (4 outputs x 4 tokens per thread) on the CUDA cores,
// followed by warp-shuffle norm reductions and a conflict-free word assembly.  All arithmetic is fp32
// with IEEE division and square root so that codes agree with the fp64 oracle except inside the 1e-5
// band around a threshold.
#include <atomic>

#include "tq_common.cuh"

namespace tq {

#ifdef TQ_TEST_HOOKS  // the cross-check kernel and its switch exist only in builds for the tests (include/tq.h)
static std::atomic<int> g_debug_quantize_fp32{0};
void debug_set_quantize_fp32(int on) { g_debug_quantize_fp32.store(on, std::memory_order_relaxed); }


__device__ __forceinline__ int swz(int k) { return ((k >> 1) * 4) & 31; }

// acc[ii][tk] += sum_k Mt[k][4 ti + ii] * xs[k][4 tt + tk]
template <int D>
__device__ __forceinline__ void gemm_tile(const float* __restrict__ Mt, const float* __restrict__ xs, int ti, int tt,
                                          float (&acc)[4][4]) {
#pragma unroll
  for (int ii = 0; ii < 4; ++ii)
#pragma unroll
    for (int tk = 0; tk < 4; ++tk) acc[ii][tk] = 0.f;
#pragma unroll 4
  for (int k = 0; k < D; ++k) {
    float4 m = *reinterpret_cast<const float4*>(Mt + k * D + 4 * ti);
    float4 x = *reinterpret_cast<const float4*>(xs + k * kTile + ((4 * tt) ^ swz(k)));
    const float mm[4] = {m.x, m.y, m.z, m.w};
    const float xx[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
      for (int tk = 0; tk < 4; ++tk) acc[ii][tk] = fmaf(mm[ii], xx[tk], acc[ii][tk]);
  }
}

// sum over the D/4 "ti" lanes that share a token group (16 lanes for D = 64, 32 for D = 128)
template <int D>
__device__ __forceinline__ float ti_sum(float v) {
#pragma unroll
  for (int o = D / 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// transposed load of a row-major [i][k] matrix into shared [k][i]
template <int D>
__device__ __forceinline__ void load_matrix_t(float* Mt, const float* __restrict__ M, int tid, int nthreads) {
  for (int idx = tid; idx < D * D; idx += nthreads) {
    int i = idx % D, k = idx / D;
    Mt[k * D + i] = M[i * D + k];
  }
}

__device__ __forceinline__ int code_of(float u, const float (&thr)[7]) {
  int c = 0;
#pragma unroll
  for (int q = 0; q < 7; ++q) c += (u > thr[q]) ? 1 : 0;
  return c;
}

// Load one tile of 32 tokens into xs[k][tok] (swizzled), applying RoPE when kIsKey.
template <int D, typename T, bool kIsKey>
__device__ __forceinline__ void load_tile(float* xs, const T* __restrict__ src /* [n_tokens][D] of this (b,h) */,
                                          const float* __restrict__ rope_cs, int tile, int start_pos, int n_tokens,
                                          int rope_layout, int tid, int nthreads) {
  constexpr int HP = D / 2;
  for (int idx = tid; idx < kTile * HP; idx += nthreads) {
    int g = idx % HP, slot = idx / HP;
    int pos = tile * kTile + slot;
    int i = pos - start_pos;
    int a = rope_layout == 0 ? 2 * g : g;
    int b = rope_layout == 0 ? 2 * g + 1 : g + HP;
    float xa = 0.f, xb = 0.f;
    if (i >= 0 && i < n_tokens) {
      xa = load_as_float<T>(src + (size_t)i * D + a);
      xb = load_as_float<T>(src + (size_t)i * D + b);
      if (kIsKey) {
        float2 cs = *reinterpret_cast<const float2*>(rope_cs + ((size_t)pos * HP + g) * 2);
        float ya = xa * cs.x - xb * cs.y;
        float yb = xa * cs.y + xb * cs.x;
        xa = ya;
        xb = yb;
      }
    }
    xs[a * kTile + (slot ^ swz(a))] = xa;
    xs[b * kTile + (slot ^ swz(b))] = xb;
  }
}

template <int D, typename T>
__global__ void __launch_bounds__(2 * D) quantize_pack_kernel(QuantArgs a) {
  using Lo = Layout<D>;
  constexpr int NT = 2 * D;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* Mk = reinterpret_cast<float*>(smem_raw);  // [D][D] PI_K^T
  float* Ms = Mk + D * D;                           // S^T
  float* Mv = Ms + D * D;                           // PI_V^T
  float* xs = Mv + D * D;                           // [D][32]
  unsigned char* cbK = reinterpret_cast<unsigned char*>(xs + D * kTile);  // [32][D] K codes
  unsigned char* cbV = cbK + kTile * D;                                    // [32][D] V codes
  unsigned char* bbK = cbV + kTile * D;                                    // [32][D] sign bits
  float* lutK = reinterpret_cast<float*>(bbK + kTile * D);                 // [8]
  float* lutV = lutK + 8;
  unsigned short* nK = reinterpret_cast<unsigned short*>(lutV + 8);  // [32]
  unsigned short* rK = nK + kTile;
  unsigned short* nV = rK + kTile;

  const int tid = threadIdx.x;
  const int ti = tid % (D / 4), tt = tid / (D / 4);
  const int bh = blockIdx.y;
  const int b = bh / a.cv.H, h = bh % a.cv.H;
  const int first_tile = a.start_pos / kTile;
  const int last_tile = (a.start_pos + a.n_tokens - 1) / kTile;
  const int tile0 = first_tile + blockIdx.x * a.tiles_per_cta;
  if (tile0 > last_tile) return;
  const int tile1 = min(last_tile, tile0 + a.tiles_per_cta - 1);

  if (blockIdx.x == 0 && h == 0 && tid == 0) a.cv.seq_len[a.layer * a.cv.B + b] = a.start_pos + a.n_tokens;

  load_matrix_t<D>(Mk, a.pi_k + (size_t)h * D * D, tid, NT);
  load_matrix_t<D>(Ms, a.S, tid, NT);
  load_matrix_t<D>(Mv, a.pi_v + (size_t)h * D * D, tid, NT);
  if (tid < 8) lutK[tid] = a.lut_k[h * 8 + tid];
  if (tid >= 32 && tid < 40) lutV[tid - 32] = a.lut_v[h * 8 + tid - 32];
  __syncthreads();
  float thrK[7], thrV[7];
#pragma unroll
  for (int q = 0; q < 7; ++q) {
    thrK[q] = 0.5f * (lutK[q] + lutK[q + 1]);
    thrV[q] = 0.5f * (lutV[q] + lutV[q + 1]);
  }

  const T* ksrc = reinterpret_cast<const T*>(a.k) + (size_t)bh * a.n_tokens * D;
  const T* vsrc = reinterpret_cast<const T*>(a.v) + (size_t)bh * a.n_tokens * D;
  const size_t unit = (size_t)a.layer * a.cv.B * a.cv.H + bh;
  unsigned char* stream = a.cv.tiles + unit * a.cv.stream_bytes;

  for (int tile = tile0; tile <= tile1; ++tile) {
    float acc[4][4];
    // ------------------------------------------------------------------ keys
    load_tile<D, T, true>(xs, ksrc, a.rope_cs, tile, a.start_pos, a.n_tokens, a.rope_layout, tid, NT);
    __syncthreads();
    gemm_tile<D>(Mk, xs, ti, tt, acc);
    __syncthreads();  // xs is about to be overwritten with the residuals
#pragma unroll
    for (int tk = 0; tk < 4; ++tk) {
      float n2 = 0.f;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) n2 = fmaf(acc[ii][tk], acc[ii][tk], n2);
      n2 = ti_sum<D>(n2);
      float n = sqrtf(n2);
      float g2 = 0.f;
      const int slot = 4 * tt + tk;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) {
        float u = n > 0.f ? acc[ii][tk] / n : 0.f;
        int c = code_of(u, thrK);
        float r = u - lutK[c];
        g2 = fmaf(r, r, g2);
        const int i = 4 * ti + ii;
        cbK[slot * D + i] = (unsigned char)c;
        xs[i * kTile + (slot ^ swz(i))] = r;
      }
      g2 = ti_sum<D>(g2);
      if (ti == 0) {
        nK[slot] = f32_to_f16_bits_clamped(n);
        rK[slot] = f32_to_f16_bits_clamped(sqrtf(g2));
      }
    }
    __syncthreads();
    gemm_tile<D>(Ms, xs, ti, tt, acc);
#pragma unroll
    for (int tk = 0; tk < 4; ++tk)
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) bbK[(4 * tt + tk) * D + 4 * ti + ii] = acc[ii][tk] >= 0.f ? 1 : 0;
    __syncthreads();
    // ------------------------------------------------------------------ values
    load_tile<D, T, false>(xs, vsrc, a.rope_cs, tile, a.start_pos, a.n_tokens, a.rope_layout, tid, NT);
    __syncthreads();
    gemm_tile<D>(Mv, xs, ti, tt, acc);
#pragma unroll
    for (int tk = 0; tk < 4; ++tk) {
      float n2 = 0.f;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) n2 = fmaf(acc[ii][tk], acc[ii][tk], n2);
      n2 = ti_sum<D>(n2);
      float n = sqrtf(n2);
      const int slot = 4 * tt + tk;
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) {
        float u = n > 0.f ? acc[ii][tk] / n : 0.f;
        cbV[slot * D + 4 * ti + ii] = (unsigned char)code_of(u, thrV);
      }
      if (ti == 0) nV[slot] = f32_to_f16_bits_clamped(n);
    }
    __syncthreads();
    // ------------------------------------------------------------------ assemble and store the tile
    // one thread per (section, word, lane) of the device tile layout (tq_common.cuh); tokens of the tile that are
    // outside this call keep their bits (read-modify-write under a mask)
    unsigned char* tp = stream + (size_t)tile * Lo::kTileBytes;
    auto in_call = [&](int slot) {
      const int pos = tile * kTile + slot;
      return pos >= a.start_pos && pos < a.start_pos + a.n_tokens;
    };
    constexpr int WTOT = 2 * Lo::KCW + Lo::KSW;
    for (int idx = tid; idx < kTile * WTOT; idx += NT) {
      const int wq = idx / kTile, lane = idx % kTile, g = lane >> 2, t = lane & 3;
      unsigned long long word = 0, mask = 0;
      auto put = [&](int bit, int nb, unsigned v) {  // bit relative to the word's first bit, may be negative
        const unsigned long long mk = (1ull << nb) - 1ull;
        if (bit <= -nb || bit >= 32) return;
        word |= bit >= 0 ? ((unsigned long long)v << bit) : ((unsigned long long)v >> (-bit));
        mask |= bit >= 0 ? (mk << bit) : (mk >> (-bit));
      };
      unsigned* p;
      if (wq < Lo::KCW) {  // K pair fields: slots g + 8 r, pairs t + 4 j
        const int w = wq;
        for (int r = 0; r < 4; ++r) {
          const int slot = g + 8 * r;
          if (!in_call(slot)) continue;
          for (int j = 0; j < Lo::J; ++j) {
            const int pr = t + 4 * j;
            put(6 * (Lo::J * r + j) - 32 * w, 6, cbK[slot * D + 2 * pr] | ((unsigned)cbK[slot * D + 2 * pr + 1] << 3));
          }
        }
        p = reinterpret_cast<unsigned*>(tp + Lo::kOffKC + word_offset(Lo::KCW, w, lane));
      } else if (wq < Lo::KCW + Lo::KSW) {  // sign bits: slots g + 8 r, sketch rows t d/4 + i
        const int w = wq - Lo::KCW;
        for (int r = 0; r < 4; ++r) {
          const int slot = g + 8 * r;
          if (!in_call(slot)) continue;
          for (int i = 0; i < D / 4; ++i) {
            const int rho = t * (D / 4) + i;
            put(sign_bit_pos<D>(slot, rho).bit - 32 * w, 1, bbK[slot * D + rho]);
          }
        }
        p = reinterpret_cast<unsigned*>(tp + Lo::kOffKS + word_offset(Lo::KSW, w, lane));
      } else {  // V codes: token pairs t + 4 j, coordinates g + 8 c
        const int w = wq - Lo::KCW - Lo::KSW;
        for (int j = 0; j < 4; ++j)
          for (int e = 0; e < 2; ++e) {
            const int slot = 2 * (t + 4 * j) + e;
            if (!in_call(slot)) continue;
            for (int c = 0; c < Lo::C; ++c) put(v_code_pos<D>(slot, g + 8 * c).bit - 32 * w, 3, cbV[slot * D + g + 8 * c]);
          }
        p = reinterpret_cast<unsigned*>(tp + Lo::kOffVC + word_offset(Lo::KCW, w, lane));
      }
      const unsigned m32 = (unsigned)mask;
      if (m32 == 0xffffffffu) *p = (unsigned)word;
      else if (m32) *p = (*p & ~m32) | ((unsigned)word & m32);
    }
    if (tid < kTile && in_call(tid)) {
      const int nl = slot_lane(tid);
      reinterpret_cast<unsigned*>(tp + Lo::kOffNK)[nl] = (unsigned)nK[tid] | ((unsigned)rK[tid] << 16);
      reinterpret_cast<unsigned short*>(tp + Lo::kOffVN)[nl] = nV[tid];
    }
    __syncthreads();
  }
}

#endif  // TQ_TEST_HOOKS

__global__ void set_seq_len_kernel(CacheView cv, int layer, int value) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < cv.B) cv.seq_len[layer * cv.B + b] = value;
}

// ---- launchers --------------------------------------------------------------------------------------------
#ifdef TQ_TEST_HOOKS
template <int D>
static size_t quant_smem_bytes() {
  return (size_t)(3 * D * D + D * kTile) * 4 + 3 * kTile * D + 16 * 4 + 3 * kTile * 2;
}

template <int D, typename T>
static cudaError_t launch_quant_t(const QuantArgs& a, int num_sms, cudaStream_t st) {
  const int first_tile = a.start_pos / kTile, last_tile = (a.start_pos + a.n_tokens - 1) / kTile;
  const int ntiles = last_tile - first_tile + 1;
  const int BH = a.cv.B * a.cv.H;
  QuantArgs b = a;
  long want = 4L * num_sms;  // aim for >= ~4 CTAs per SM worth of work items
  int tpc = (int)(((long)ntiles * BH + want - 1) / want);
  b.tiles_per_cta = tpc < 1 ? 1 : (tpc > 16 ? 16 : tpc);
  dim3 grid((ntiles + b.tiles_per_cta - 1) / b.tiles_per_cta, BH);
  size_t smem = quant_smem_bytes<D>();
  cudaError_t e = cudaFuncSetAttribute(quantize_pack_kernel<D, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  quantize_pack_kernel<D, T><<<grid, 2 * D, smem, st>>>(b);
  count_launch();
  return cudaGetLastError();
}

#endif  // TQ_TEST_HOOKS

cudaError_t launch_quantize_pack(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st) {
  if (a.n_tokens == 0) {
    set_seq_len_kernel<<<(a.cv.B + 127) / 128, 128, 0, st>>>(a.cv, a.layer, a.start_pos);
    count_launch();
    return cudaGetLastError();
  }
  // the tensor-core kernel (tq_quantize_tc.cu) is the product path
#ifdef TQ_TEST_HOOKS
  // tq_debug_set_quantize_impl(1) selects the CUDA-core kernel of this file (it only knows the default residual mode)
  if (g_debug_quantize_fp32.load(std::memory_order_relaxed) != 0 && !a.literal && !a.cv.vsk) {
    if (D == 64) return dt == TQ_F16 ? launch_quant_t<64, __half>(a, num_sms, st) : launch_quant_t<64, float>(a, num_sms, st);
    return dt == TQ_F16 ? launch_quant_t<128, __half>(a, num_sms, st) : launch_quant_t<128, float>(a, num_sms, st);
  }
#endif
  return launch_quantize_pack_tc(a, D, dt, num_sms, st);
}

}  // namespace tq
