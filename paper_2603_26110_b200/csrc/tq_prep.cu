// tq_prep.cu — the small kernel in front of the streaming decode kernel.
//
// One CTA per (layer-in-call, head, run of up to 32 batch entries) does, depending on the template flags,
//   kAppend : quantize-and-pack ONE new token per batch entry (PAPER.md:111-116 per vector;
//             BASELINE.json:configs[2]): RoPE(k) -> PI_K -> norm, codes, residual -> S r -> bits;
//             PI_V v -> norm, codes; the pieces are written into the tile slot seq_len[layer][b] (device tile layout,
//             tq_common.cuh) and the last head of the batch entry to arrive bumps seq_len;
//   kQuery  : query preparation for the fused decode kernel (Eq. 4 moves PI to the query; north_star):
//             q'' = PI_K RoPE(q), z = S q''  -> the decode kernel's MMA operands in the workspace (FragLayout), pre-scaled
//             so that logits come out in log2 units; plus the head's fp16 dequantisation tables.
// tq_append = <true,false>, tq_decode_attn = <false,true>, tq_decode_step / tq_decode_model_step = <true,true>.
//
// For the batch entries of one head the five d x d mat-vecs are two small GEMMs, [k; q; v rows] x PI^T and
// [r; q'' rows] x S^T: they run on mma.sync.m16n8k16 with the same exactness scheme as the tcgen05 prefill kernel
// (tq_quantize_tc.cu): fp16 two-term splits a = a_hi + a_lo of both operands, D = A_hi B_hi + A_lo B_hi + A_hi B_lo with
// fp32 accumulation, power-of-two scalings that cancel exactly (PI x16, vectors by 2^-exponent(max |x|), r x8).  A warp
// owns d/64 n-tiles (8 matrix rows each) and reads their B fragments straight from global memory (L2), so no matrix is
// staged.  Everything per entry (RoPE, maxima, norms, codes, residual, operand splits) is done by one warp per entry with
// shuffles: six CTA barriers in all, whatever the number of entries.  (A first version kept matrix rows in registers and
// used CUDA-core FMAs, two of six warps at a time: 190 us for the 33-layer step; profiles/r02_prep.md.)
#include "tq_common.cuh"

namespace tq {

struct PrepArgs {
  CacheView cv;
  const float *pi_k, *pi_v, *lut_k, *lut_v, *S, *rope_cs;  // full [L][H]... arrays
  const void *q, *k, *v;                                    // [Lc][B][H][D] each (k, v: append; q: query)
  void* out;                                                // [Lc][B][H][D] (zeroed here for empty caches)
  const int32_t* q_pos;                                     // [Lc][B] or nullptr
  unsigned* frags;                                          // workspace [units][FragLayout<D>::kWords]
  unsigned* tabs;                                           // workspace [layers_call * H][kTabWords]
  int layer_begin, rope_layout;
  int literal;          // paper-literal Eq. 6-7 mode of the append (include/tq.h)
  const float* ebar_k;  // [L][H]
};

constexpr int kPrepThreads = 256;
constexpr int kPrepWarps = kPrepThreads / 32;

// EB = batch entries per CTA: 32 (two 16-row m-tiles per operand block; the multi-layer model step, where the instruction
// count per SM matters) or 8 (k and q rows share one m-tile; a single layer, where the latency of one CTA matters)
template <int D, int EB>
struct PrepCfg {
  static constexpr int HP = D + 8;   // row pitch of the fp16 operand rows, in halves: A-fragment reads are conflict free
  static constexpr int FP = D + 8;   // row pitch of the fp32 result rows
  static constexpr int ROWS = EB == 8 ? 32 : 3 * EB;  // operand rows: [0, EB) k then r | [EB, 2 EB) q then q'' | [2 EB, 3 EB) v
  static constexpr size_t kSmemBytes = (size_t)2 * ROWS * HP * 2 /* hi, lo */ + (size_t)ROWS * FP * 4 /* results */ +
                                       (size_t)2 * EB * D /* cK, cV */;
};

__device__ __forceinline__ void mma16816p(float (&d)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0, unsigned b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// (x0, x1) -> fp16 pairs hi and lo with x = hi + lo
__device__ __forceinline__ void split_pair(float x0, float x1, unsigned& hi, unsigned& lo) {
  const __half2 h = __floats2half2_rn(x0, x1);
  const float2 hf = __half22float2(h);
  const __half2 l = __floats2half2_rn(x0 - hf.x, x1 - hf.y);
  hi = *reinterpret_cast<const unsigned*>(&h);
  lo = *reinterpret_cast<const unsigned*>(&l);
}
// 2^-e and 2^e with 2^e <= amax < 2^(e+1) (1, 1 for zero / denormal amax)
__device__ __forceinline__ void pow2_scale_p(float amax, float& s, float& inv_s) {
  unsigned E = (__float_as_uint(amax) >> 23) & 0xffu;
  E = E < 2u ? 127u : (E > 252u ? 252u : E);
  s = __uint_as_float((254u - E) << 23);
  inv_s = __uint_as_float(E << 23);
}
__device__ __forceinline__ int code_of7(float u, const float* lut) {
  int c = 0;
#pragma unroll
  for (int q = 0; q < 7; ++q) c += (u > 0.5f * (lut[q] + lut[q + 1])) ? 1 : 0;
  return c;
}

template <int HPITCH>
struct PitchCfg {
  static constexpr int HP = HPITCH, FP = HPITCH;
};

// C[rows m0 .. m0 + 16 MT) x [n-tile rows n0 .. n0 + 8) = A (fp16 hi / lo rows in shared memory) x M^T, M fp32 row-major in
// global memory scaled by mscale; the accumulators are multiplied by rscale[row] and stored as fp32 rows.
template <int D, int HPITCH, int MT, bool kLoTermA>
__device__ __forceinline__ void gemm_rows(const __half* Ah, const __half* Al, int m0, const float* __restrict__ M, float mscale, int n0,
                                          float* C, const float* rscale, int lane) {
  using Cfg = PitchCfg<HPITCH>;
  const int g = lane >> 2, t = lane & 3;
  float acc[MT][4];
#pragma unroll
  for (int i = 0; i < MT; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
  // B fragments of this n-tile for every k-step: M[n0 + g][16 ks + 2 t + {0, 1, 8, 9}]
  float2 bf[D / 16][2];
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks) {
    bf[ks][0] = __ldg(reinterpret_cast<const float2*>(M + (size_t)(n0 + g) * D + 16 * ks + 2 * t));
    bf[ks][1] = __ldg(reinterpret_cast<const float2*>(M + (size_t)(n0 + g) * D + 16 * ks + 2 * t + 8));
  }
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks) {
    unsigned bh0, bl0, bh1, bl1;
    split_pair(bf[ks][0].x * mscale, bf[ks][0].y * mscale, bh0, bl0);
    split_pair(bf[ks][1].x * mscale, bf[ks][1].y * mscale, bh1, bl1);
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
      const int r0 = m0 + 16 * mt + g;
      const unsigned* ph = reinterpret_cast<const unsigned*>(Ah + (size_t)r0 * Cfg::HP + 16 * ks + 2 * t);
      const unsigned* ph8 = reinterpret_cast<const unsigned*>(Ah + (size_t)(r0 + 8) * Cfg::HP + 16 * ks + 2 * t);
      const unsigned a0 = ph[0], a1 = ph8[0], a2 = ph[4], a3 = ph8[4];
      mma16816p(acc[mt], a0, a1, a2, a3, bh0, bh1);
      mma16816p(acc[mt], a0, a1, a2, a3, bl0, bl1);
      if (kLoTermA) {
        const unsigned* pl = reinterpret_cast<const unsigned*>(Al + (size_t)r0 * Cfg::HP + 16 * ks + 2 * t);
        const unsigned* pl8 = reinterpret_cast<const unsigned*>(Al + (size_t)(r0 + 8) * Cfg::HP + 16 * ks + 2 * t);
        mma16816p(acc[mt], pl[0], pl8[0], pl[4], pl8[4], bh0, bh1);
      }
    }
  }
#pragma unroll
  for (int mt = 0; mt < MT; ++mt) {
    const int r0 = m0 + 16 * mt + g;
    const float s0 = rscale[r0], s1 = rscale[r0 + 8];
    *reinterpret_cast<float2*>(C + (size_t)r0 * Cfg::FP + n0 + 2 * t) = make_float2(acc[mt][0] * s0, acc[mt][1] * s0);
    *reinterpret_cast<float2*>(C + (size_t)(r0 + 8) * Cfg::FP + n0 + 2 * t) = make_float2(acc[mt][2] * s1, acc[mt][3] * s1);
  }
}

template <int D, typename T, bool kAppend, bool kQuery, int EB>
__global__ void __launch_bounds__(kPrepThreads) prep_kernel(PrepArgs a) {
  using Lo = Layout<D>;
  using Cfg = PrepCfg<D, EB>;
  using FL = FragLayout<D>;
  constexpr int NT = kPrepThreads, NW = kPrepWarps;
  constexpr int HPAIR = D / 2;      // RoPE pairs per vector
  constexpr int PL = D / 64;        // RoPE pairs per lane
  constexpr float kInvSqrtD = D == 64 ? 0.125f : 0.08838834764831845f;
  constexpr float kScaleK = 1.4426950408889634f * kInvSqrtD;             // log2(e) / sqrt(d)
  constexpr float kScaleS = kScaleK * 1.2533141373155003f / (float)D;  // ... * sqrt(pi/2) / m, m = D
  constexpr bool kValLo = sizeof(T) == 4;  // fp16 values are exact operands: no lo term
  extern __shared__ __align__(16) unsigned char dsm[];
  __half* Ah = reinterpret_cast<__half*>(dsm);                          // [ROWS][HP] hi parts
  __half* Al = Ah + (size_t)Cfg::ROWS * Cfg::HP;                        // lo parts
  float* Y = reinterpret_cast<float*>(Al + (size_t)Cfg::ROWS * Cfg::HP);  // [ROWS][FP]: y_k | q'' | y_v, then S r | z
  unsigned char (*cK)[D] = reinterpret_cast<unsigned char (*)[D]>(Y + (size_t)Cfg::ROWS * Cfg::FP);
  unsigned char (*cV)[D] = cK + EB;
  __shared__ float rscale[Cfg::ROWS];  // accumulator -> result, per operand row
  __shared__ float nrm[4][EB];         // |k|, |r_k|, |v|, |r_v| of the appended token
  __shared__ float qsc[EB][2];         // 2^eq (scaling of the q'' operand rows), reserved
  __shared__ float lutK[8], lutV[8];
  __shared__ int s_len0[EB], s_full[EB];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int B = a.cv.B, H = a.cv.H;
  const int nrun = (B + EB - 1) / EB;
  const int run = (int)blockIdx.x % nrun, lh_c = (int)blockIdx.x / nrun;  // (layer-in-call, head), run of batch entries
  const int lc = lh_c / H, h = lh_c % H;
  const int layer = a.layer_begin + lc;
  const int b0 = run * EB, nb = min(EB, B - b0);
  const int mt_n = nb > 16 ? 2 : 1;  // m-tiles that hold entries (EB = 32)
  const size_t lh = (size_t)layer * H + h;
  auto unit_of = [&](int e) { return ((size_t)lc * B + b0 + e) * H + h; };        // unit inside the call (q, k, v, out, operands)
  auto stream_of = [&](int e) { return ((size_t)layer * B + b0 + e) * H + h; };  // unit inside the cache

  const bool vsk = kAppend && a.cv.vsk != nullptr;  // V-side sketch (tq_shape.v_qjl = 1)
  pdl_trigger();  // the streaming kernel behind this one may be scheduled
  if constexpr (EB == 8) {  // rows [24, 32) pad the value block to a whole m-tile
    for (int idx = tid; idx < 8 * Cfg::HP / 2; idx += NT) {
      reinterpret_cast<unsigned*>(Ah + (size_t)24 * Cfg::HP)[idx] = 0u;
      reinterpret_cast<unsigned*>(Al + (size_t)24 * Cfg::HP)[idx] = 0u;
    }
    if (tid < 8) rscale[24 + tid] = 0.f;
  }
  if (tid < 8) lutK[tid] = a.lut_k[lh * 8 + tid];
  if (tid >= 32 && tid < 40) lutV[tid - 32] = a.lut_v[lh * 8 + tid - 32];
  // ---- the cache lengths first: the RoPE positions and the target tile slots hang off them.  (The length of an entry
  //      cannot change while its heads are still arriving.)
  if (tid >= 64 && tid < 64 + EB) {
    const int e = tid - 64;
    const int len0 = e < nb ? __ldcg(a.cv.seq_len + layer * B + b0 + e) : 0;
    s_len0[e] = len0;
    s_full[e] = kAppend && len0 >= a.cv.max_seq;
  }
  __syncthreads();

  // ---- the store stage at the end: a warp owns entries warp, warp + 8, ... (EPW of them) and makes four passes over
  //      them with lane = (entry n, piece): K blocks (4 per entry), sign bytes (8 U), V blocks (8, read-modify-write: a V
  //      field is shared with the other token of the pair, appended by an earlier call), norms (1).  The V halfwords are
  //      requested here, long before they are needed.
  constexpr int HW = 3 * D / 64;       // halfwords per (lane, token) block of K fields, and per (lane, token pair) block of V fields
  constexpr int EPW = EB / NW;         // entries per warp in the store stage
  unsigned short vold[HW];
#pragma unroll
  for (int hw = 0; hw < HW; ++hw) vold[hw] = 0;
  if (kAppend && lane < 8 * EPW) {
    const int e = warp + (lane >> 3) * NW, gi = lane & 7;
    if (e < nb && s_len0[e] < a.cv.max_seq) {
      const int len = s_len0[e], slot = len % kTile, pp = slot >> 1;
      const unsigned char* tp = a.cv.tiles + stream_of(e) * a.cv.stream_bytes + (size_t)(len / kTile) * Lo::kTileBytes;
#pragma unroll
      for (int hw = 0; hw < HW; ++hw) {
        const int hidx = (pp >> 2) * HW + hw;  // halfword of lane (gi, pp & 3)'s V string
        vold[hw] = __ldcg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffVC + word_offset(Lo::KCW, hidx >> 1, 4 * gi + (pp & 3))) +
                          (hidx & 1));
      }
    }
  }

  // ---- stage 1: one warp per (entry, vector): load, RoPE, 2^-exponent(max) scaling, fp16 hi / lo operand rows.
  //      Lane l owns RoPE pairs l + 32 j.  The loads of kTB tasks are issued before the first one is used (a task is one
  //      DRAM round trip; a warp has twelve of them).
  constexpr int NVEC = (kAppend ? 2 : 0) + (kQuery ? 1 : 0);  // k, v | q
  constexpr int NTASK = EB * NVEC / NW;                        // tasks per warp: 12 | 8 | 4 (EB = 32), 3 | 2 | 1 (EB = 8)
  constexpr int kTB = NTASK <= 4 ? NTASK : ((D == 64 && NTASK == 12) ? 6 : 4);
  static_assert(NTASK % kTB == 0, "whole batches");
  for (int tb0 = 0; tb0 < NTASK; tb0 += kTB) {
    float xa[kTB][PL], xb[kTB][PL];
    float2 cs[kTB][PL];
#pragma unroll
    for (int q = 0; q < kTB; ++q) {
      const int task = warp + (tb0 + q) * NW, e = task % EB;
      const int vec = (!kAppend) ? 2 : (task / EB == 0 ? 0 : (task / EB == 1 ? 1 : 2));  // 0 = k, 1 = v, 2 = q
#pragma unroll
      for (int j = 0; j < PL; ++j) xa[q][j] = xb[q][j] = 0.f, cs[q][j] = make_float2(1.f, 0.f);
      if (e < nb) {
        const T* src = reinterpret_cast<const T*>(vec == 0 ? a.k : (vec == 1 ? a.v : a.q)) + unit_of(e) * D;
        const int len0 = s_len0[e];
        int pos = 0;
        if (vec == 0) pos = min(len0, a.cv.max_seq - 1);  // the appended key sits at index len0
        if (vec == 2) {                                    // the query defaults to the newest cached token
          const int len1 = (kAppend && !s_full[e]) ? len0 + 1 : len0;
          pos = a.q_pos ? a.q_pos[lc * B + b0 + e] : len1 - 1;
          pos = max(0, min(pos, a.cv.max_seq - 1));
          if (len1 <= 0) {  // empty cache: no tile for this unit in the streaming kernel, out = 0
            T* outp = reinterpret_cast<T*>(a.out) + unit_of(e) * D;
            for (int i = lane; i < D; i += 32) {
              if constexpr (sizeof(T) == 2) outp[i] = __float2half_rn(0.f);
              else outp[i] = 0.f;
            }
          }
        }
#pragma unroll
        for (int j = 0; j < PL; ++j) {
          const int gp = lane + 32 * j;
          const bool adj = vec == 1 || a.rope_layout == 0;
          const int ia = adj ? 2 * gp : gp, ib = adj ? 2 * gp + 1 : gp + HPAIR;
          xa[q][j] = load_as_float<T>(src + ia), xb[q][j] = load_as_float<T>(src + ib);
          if (vec != 1) cs[q][j] = __ldg(reinterpret_cast<const float2*>(a.rope_cs + ((size_t)pos * HPAIR + gp) * 2));
        }
      }
    }
#pragma unroll
    for (int q = 0; q < kTB; ++q) {
      const int task = warp + (tb0 + q) * NW, e = task % EB;
      const int vec = (!kAppend) ? 2 : (task / EB == 0 ? 0 : (task / EB == 1 ? 1 : 2));
      const int orow = vec == 0 ? e : (vec == 2 ? EB + e : 2 * EB + e);
      float amax = 0.f;
#pragma unroll
      for (int j = 0; j < PL; ++j) {
        amax = fmaxf(amax, fmaxf(fabsf(xa[q][j]), fabsf(xb[q][j])));
        const float ya = xa[q][j] * cs[q][j].x - xb[q][j] * cs[q][j].y, yb = xa[q][j] * cs[q][j].y + xb[q][j] * cs[q][j].x;
        xa[q][j] = ya, xb[q][j] = yb;
      }
      amax = warp_max(amax);
      float sc, inv_s;
      pow2_scale_p(amax, sc, inv_s);  // |RoPE(x) s| < 2 sqrt 2
      if (lane == 0) rscale[orow] = inv_s * 0.0625f;  // y = 16 s PI x
#pragma unroll
      for (int j = 0; j < PL; ++j) {
        const int gp = lane + 32 * j;
        const bool adj = vec == 1 || a.rope_layout == 0;
        const int ia = adj ? 2 * gp : gp, ib = adj ? 2 * gp + 1 : gp + HPAIR;
        if (adj) {
          unsigned hi, lo;
          split_pair(xa[q][j] * sc, xb[q][j] * sc, hi, lo);
          *reinterpret_cast<unsigned*>(Ah + (size_t)orow * Cfg::HP + ia) = hi;
          *reinterpret_cast<unsigned*>(Al + (size_t)orow * Cfg::HP + ia) = lo;
        } else {
          const __half ha = __float2half_rn(xa[q][j] * sc), hb = __float2half_rn(xb[q][j] * sc);
          Ah[(size_t)orow * Cfg::HP + ia] = ha, Ah[(size_t)orow * Cfg::HP + ib] = hb;
          Al[(size_t)orow * Cfg::HP + ia] = __float2half_rn(xa[q][j] * sc - __half2float(ha));
          Al[(size_t)orow * Cfg::HP + ib] = __float2half_rn(xb[q][j] * sc - __half2float(hb));
        }
      }
    }
  }
  __syncthreads();

  // ---- stage 2: [k rows; q rows] x PI_K^T and [v rows] x PI_V^T: a warp owns n-tiles warp, warp + 8, ...
  //      product over the k / q row blocks with matrix M (EB = 8: both blocks are one m-tile)
  auto kq_product = [&](const float* M, float mscale, int n0) {
    constexpr int HPI = Cfg::HP;
    if constexpr (EB == 8) {
      gemm_rows<D, HPI, 1, true>(Ah, Al, 0, M, mscale, n0, Y, rscale, lane);
    } else if (kAppend && kQuery) {
      if (mt_n == 2) gemm_rows<D, HPI, 4, true>(Ah, Al, 0, M, mscale, n0, Y, rscale, lane);
      else {
        gemm_rows<D, HPI, 1, true>(Ah, Al, 0, M, mscale, n0, Y, rscale, lane);
        gemm_rows<D, HPI, 1, true>(Ah, Al, EB, M, mscale, n0, Y, rscale, lane);
      }
    } else {
      const int m0 = kAppend ? 0 : EB;
      if (mt_n == 2) gemm_rows<D, HPI, 2, true>(Ah, Al, m0, M, mscale, n0, Y, rscale, lane);
      else gemm_rows<D, HPI, 1, true>(Ah, Al, m0, M, mscale, n0, Y, rscale, lane);
    }
  };
  for (int nt = warp; nt < D / 8; nt += NW) {
    kq_product(a.pi_k + lh * D * D, 16.f, 8 * nt);
    if (kAppend) {
      const float* Pv = a.pi_v + lh * D * D;
      if (EB == 8 || mt_n == 1) gemm_rows<D, Cfg::HP, 1, kValLo>(Ah, Al, 2 * EB, Pv, 16.f, 8 * nt, Y, rscale, lane);
      else gemm_rows<D, Cfg::HP, 2, kValLo>(Ah, Al, 2 * EB, Pv, 16.f, 8 * nt, Y, rscale, lane);
    }
  }
  __syncthreads();

  // ---- stage 3: one warp per (entry, vector): norms, codes, residual; operand rows of the sketch product
  //      (rows [0, 32): r x 8; rows [32, 64): q'' 2^eq, which are also the decode kernel's q operand)
  for (int task = warp; task < EB * NVEC; task += NW) {
    const int e = task % EB;
    const int vec = (!kAppend) ? 2 : (task / EB == 0 ? 0 : (task / EB == 1 ? 1 : 2));
    const int yrow = vec == 0 ? e : (vec == 2 ? EB + e : 2 * EB + e);
    if (e >= nb) continue;  // padding rows stay zero
    const float* y = Y + (size_t)yrow * Cfg::FP;
    float2 v2[PL];
#pragma unroll
    for (int j = 0; j < PL; ++j) v2[j] = *reinterpret_cast<const float2*>(y + 2 * (lane + 32 * j));
    if (vec == 2) {  // q'': power-of-two scaling that puts max |q''| 2^eq in [2^13, 2^14), hi / lo rows
      float qm = 0.f;
#pragma unroll
      for (int j = 0; j < PL; ++j) qm = fmaxf(qm, fmaxf(fabsf(v2[j].x), fabsf(v2[j].y)));
      qm = warp_max(qm);
      const int E = (int)((__float_as_uint(qm) >> 23) & 0xffu);
      const int eq = 13 - ((E == 0 || E == 255) ? 0 : E - 127);
      const float sq = __uint_as_float((unsigned)(max(-100, min(100, eq)) + 127) << 23);
#pragma unroll
      for (int j = 0; j < PL; ++j) {
        unsigned hi, lo;
        split_pair(v2[j].x * sq, v2[j].y * sq, hi, lo);
        *reinterpret_cast<unsigned*>(Ah + (size_t)yrow * Cfg::HP + 2 * (lane + 32 * j)) = hi;
        *reinterpret_cast<unsigned*>(Al + (size_t)yrow * Cfg::HP + 2 * (lane + 32 * j)) = lo;
      }
      if (lane == 0) {
        rscale[yrow] = 1.f / sq;  // z = S q'': undo 2^eq (exact)
        qsc[e][0] = 1.f / sq;
      }
      continue;
    }
    float n2 = 0.f;
#pragma unroll
    for (int j = 0; j < PL; ++j) n2 = fmaf(v2[j].x, v2[j].x, fmaf(v2[j].y, v2[j].y, n2));
    n2 = warp_sum(n2);
    const float n = a.literal ? 1.f : sqrtf(n2);                  // literal mode: the activation itself is coded
    const float inv = a.literal ? 1.f : (n > 0.f ? 1.0f / n : 0.f);
    const float* lut = vec == 0 ? lutK : lutV;
    // residual operand scale: 8 for a unit vector; in literal mode a power of two that keeps r inside the fp16 range
    float rsc = 8.f;
    if (a.literal && vec == 0) {
      float rm = 0.f;
#pragma unroll
      for (int j = 0; j < PL; ++j) {
        rm = fmaxf(rm, fmaxf(fabsf(v2[j].x - lut[code_of7(v2[j].x, lut)]), fabsf(v2[j].y - lut[code_of7(v2[j].y, lut)])));
      }
      rm = warp_max(rm);
      float inv_r;
      pow2_scale_p(rm, rsc, inv_r);
    }
    float g2 = 0.f;
#pragma unroll
    for (int j = 0; j < PL; ++j) {
      const int i0 = 2 * (lane + 32 * j);
      const float u0 = v2[j].x * inv, u1 = v2[j].y * inv;
      const int c0 = code_of7(u0, lut), c1 = code_of7(u1, lut);
      if (vec == 0) {
        const float r0 = u0 - lut[c0], r1 = u1 - lut[c1];
        g2 = fmaf(r0, r0, fmaf(r1, r1, g2));
        cK[e][i0] = (unsigned char)c0, cK[e][i0 + 1] = (unsigned char)c1;
        unsigned hi, lo;
        split_pair(r0 * rsc, r1 * rsc, hi, lo);  // only sign(S r) is used
        *reinterpret_cast<unsigned*>(Ah + (size_t)yrow * Cfg::HP + i0) = hi;
        *reinterpret_cast<unsigned*>(Al + (size_t)yrow * Cfg::HP + i0) = lo;
      } else {
        cV[e][i0] = (unsigned char)c0, cV[e][i0 + 1] = (unsigned char)c1;
        if (vsk) {  // V-side sketch: the residual of the value becomes an operand row of the S product too
          const float r0 = u0 - lut[c0], r1 = u1 - lut[c1];
          g2 = fmaf(r0, r0, fmaf(r1, r1, g2));
          unsigned hi, lo;
          split_pair(r0 * 8.f, r1 * 8.f, hi, lo);
          *reinterpret_cast<unsigned*>(Ah + (size_t)yrow * Cfg::HP + i0) = hi;
          *reinterpret_cast<unsigned*>(Al + (size_t)yrow * Cfg::HP + i0) = lo;
        }
      }
    }
    if (vec == 0) {
      g2 = warp_sum(g2);
      if (lane == 0) nrm[0][e] = n, nrm[1][e] = sqrtf(g2), rscale[yrow] = 1.f;
    } else {
      if (vsk) g2 = warp_sum(g2);
      if (lane == 0) {
        nrm[2][e] = n;
        if (vsk) nrm[3][e] = sqrtf(g2), rscale[yrow] = 1.f;
      }
    }
  }
  __syncthreads();

  // ---- stage 4: [r rows; q'' rows] x S^T -> sign bits | z   (and the value residual rows with the V-side sketch)
  for (int nt = warp; nt < D / 8; nt += NW) {
    kq_product(a.S, 1.f, 8 * nt);
    if (kAppend && vsk) {
      if (EB == 8 || mt_n == 1) gemm_rows<D, Cfg::HP, 1, true>(Ah, Al, 2 * EB, a.S, 1.f, 8 * nt, Y, rscale, lane);
      else gemm_rows<D, Cfg::HP, 2, true>(Ah, Al, 2 * EB, a.S, 1.f, 8 * nt, Y, rscale, lane);
    }
  }
  __syncthreads();

  if (kQuery) {
    // ---- the decode kernel's operands (tq_common.cuh FragLayout), one warp per entry.  The q words are the q'' 2^eq
    //      operand rows as they stand (kscale = 2^-eq log2(e)/sqrt(d)); z = S q'' is scaled to max |z_s| 2^ez in
    //      [2^13, 2^14) and split per sketch row with the fragment's 2^-p weights.
    for (int e = warp; e < nb; e += NW) {
      const float* z = Y + (size_t)(EB + e) * Cfg::FP;
      float zm = 0.f, zsum = 0.f;
#pragma unroll
      for (int i = lane; i < D; i += 32) {
        const float zv = z[i] * kScaleS;
        zm = fmaxf(zm, fabsf(zv));
        zsum += zv;
      }
      zm = warp_max(zm), zsum = warp_sum(zsum);
      const int E = (int)((__float_as_uint(zm) >> 23) & 0xffu);
      const int ez = 13 - ((E == 0 || E == 255) ? 0 : E - 127);
      auto p2 = [](int ee) { return __uint_as_float((unsigned)(max(-100, min(100, ee)) + 127) << 23); };
      unsigned* fb = a.frags + unit_of(e) * FL::kWords;
      const __half* qh = Ah + (size_t)(EB + e) * Cfg::HP;
      const __half* ql = Al + (size_t)(EB + e) * Cfg::HP;
      for (int wi = lane; wi < FL::kScalOff; wi += 32) {
        const int pat = wi / FL::kWordsPerPat, wd = wi % FL::kWordsPerPat, t = pat & 3;
        const bool lo = pat >> 2;
        unsigned word;
        if (wd < 2 * FL::KS) {
          const int c0 = 16 * (wd >> 1) + 2 * t + 8 * (wd & 1);
          word = *reinterpret_cast<const unsigned*>((lo ? ql : qh) + c0);
        } else {
          const int ks = (wd - 2 * FL::KS) >> 1, reg = wd & 1, p0 = 2 * (ks & 3);
          const int rho = t * (D / 4) + 16 * (ks >> 2) + p0 + reg;
          const float sc = kScaleS * p2(ez - p0 - reg);
          unsigned hi, lw;
          split_pair(z[rho] * sc, z[rho + 8] * sc, hi, lw);
          word = lo ? lw : hi;
        }
        fb[wi] = word;
      }
      if (lane == 0) {
        float* sc = reinterpret_cast<float*>(fb + FL::kScalOff);
        sc[0] = qsc[e][0] * kScaleK, sc[1] = p2(25 - ez), sc[2] = zsum, sc[3] = 0.f;
      }
    }
    if (tid < 64 && run == 0) {  // the head's dequantisation tables
      auto pair16 = [](float x0, float x1, bool lo) {
        unsigned hi, lw;
        split_pair(x0, x1, hi, lw);
        return lo ? lw : hi;
      };
      const int c0 = tid & 7, c1 = tid >> 3;
      unsigned* tb = a.tabs + (size_t)lh_c * kTabWords;
      tb[tid] = pair16(lutK[c0], lutK[c1], false);
      tb[64 + tid] = pair16(lutK[c0], lutK[c1], true);
      tb[128 + tid] = pair16(lutV[c0], lutV[c1], false);
      tb[192 + tid] = pair16(lutV[c0], lutV[c1], true);
      if (tid == 0) {
        bool exact = true;
#pragma unroll
        for (int i = 0; i < 8; ++i)
          exact = exact && __half2float(__float2half_rn(lutK[i])) == lutK[i] && __half2float(__float2half_rn(lutV[i])) == lutV[i];
        tb[256] = exact ? 1u : 0u;
      }
    }
  }
  if (!kAppend) return;

  // ---- stage 5 (append): the four store passes (see above)
  auto tile_of = [&](int e, int& slot) {
    const int len = s_len0[e];
    slot = len % kTile;
    return a.cv.tiles + stream_of(e) * a.cv.stream_bytes + (size_t)(len / kTile) * Lo::kTileBytes;
  };
  if (lane < 4 * EPW) {  // K: pairs t + 4 j, field j at bit 6 j of the block
    const int e = warp + (lane >> 2) * NW, t = lane & 3;
    if (e < nb && !s_full[e]) {
      int slot;
      unsigned char* tp = tile_of(e, slot);
      const int g = slot & 7, r = slot >> 3;
      unsigned long long lo = 0ull, hi = 0ull;
#pragma unroll
      for (int j = 0; j < Lo::J; ++j) {
        const int p = t + 4 * j;
        const unsigned long long f = (unsigned)(cK[e][2 * p] | (cK[e][2 * p + 1] << 3));
        const int bit = 6 * j;
        if (bit < 64) lo |= f << bit;
        if (bit + 6 > 64) hi |= bit >= 64 ? f << (bit - 64) : f >> (64 - bit);
      }
#pragma unroll
      for (int hw = 0; hw < HW; ++hw) {
        const int hidx = r * HW + hw;
        const unsigned short v = (unsigned short)(hw < 4 ? lo >> (16 * hw) : hi >> (16 * (hw - 4)));
        reinterpret_cast<unsigned short*>(tp + Lo::kOffKC + word_offset(Lo::KCW, hidx >> 1, 4 * g + t))[hidx & 1] = v;
      }
    }
  }
  for (int item = lane; item < 8 * Lo::U * EPW; item += 32) {  // sign bytes: bit k = [(S r)_rho >= 0], rho = t d/4 + 16 u + 8 hb + k
    const int e = warp + (item / (8 * Lo::U)) * NW, si = item % (8 * Lo::U);
    if (e < nb && !s_full[e]) {
      int slot;
      unsigned char* tp = tile_of(e, slot);
      const int g = slot & 7, r = slot >> 3;
      const int t = si / (2 * Lo::U), u = (si / 2) % Lo::U, hb = si & 1;
      const float* sr = Y + (size_t)e * Cfg::FP + t * (D / 4) + 16 * u + 8 * hb;
      unsigned v = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) v |= (sr[k] >= 0.f ? 1u : 0u) << k;
      const int word = (slot >> 4) * Lo::U + u, byte = 2 * hb + (r & 1);
      *(tp + Lo::kOffKS + word_offset(Lo::KSW, word, 4 * g + t) + byte) = (unsigned char)v;
    }
  }
  if (lane < 8 * EPW) {  // V: coordinates gi + 8 c, three-bit slices at 6 c + 3 (slot & 1)
    const int e = warp + (lane >> 3) * NW, gi = lane & 7;
    if (e < nb && !s_full[e]) {
      int slot;
      unsigned char* tp = tile_of(e, slot);
      const int pp = slot >> 1, sh0 = 3 * (slot & 1);
      unsigned long long lo = 0ull, hi = 0ull, mlo = 0ull, mhi = 0ull;
#pragma unroll
      for (int c = 0; c < Lo::C; ++c) {
        const unsigned long long f = cV[e][gi + 8 * c], m7 = 7ull;
        const int bit = 6 * c;
        if (bit + 6 <= 64) lo |= f << (bit + sh0), mlo |= m7 << (bit + sh0);
        else if (bit >= 64) hi |= f << (bit - 64 + sh0), mhi |= m7 << (bit - 64 + sh0);
        else {  // field 10 of d = 128 covers bits [60, 66)
          const unsigned long long f6 = f << sh0, m6 = m7 << sh0;
          lo |= f6 << bit, mlo |= m6 << bit;
          hi |= f6 >> (64 - bit), mhi |= m6 >> (64 - bit);
        }
      }
#pragma unroll
      for (int hw = 0; hw < HW; ++hw) {
        const int hidx = (pp >> 2) * HW + hw;
        const unsigned short v = (unsigned short)(hw < 4 ? lo >> (16 * hw) : hi >> (16 * (hw - 4)));
        const unsigned short mk = (unsigned short)(hw < 4 ? mlo >> (16 * hw) : mhi >> (16 * (hw - 4)));
        unsigned short* vptr = reinterpret_cast<unsigned short*>(tp + Lo::kOffVC + word_offset(Lo::KCW, hidx >> 1, 4 * gi + (pp & 3))) + (hidx & 1);
        *vptr = (unsigned short)((vold[hw] & ~mk) | v);
      }
    }
  }
  if (vsk) {
    // V-side sketch tile: the token's bit of sketch row rho sits in lane (rho & 7, t of the slot), word ks (D/64) + (mt >> 2),
    // bit 16 e + 4 (mt & 3) + 2 rh + th: one lane per (g, word) clears the token's eight bits of that word and sets the new ones
    using Vs = VskLayout<D>;
    constexpr int WPT = 8 * (D / 64);  // words a token touches
    for (int k = 0; k < EPW; ++k) {
      const int e = warp + k * NW;
      if (e >= nb || s_full[e] || lane >= WPT) continue;
      const int len = s_len0[e], slot = len % kTile;
      unsigned char* vt = a.cv.vsk + stream_of(e) * a.cv.vsk_stream_bytes + (size_t)(len / kTile) * Vs::kTileBytes;
      const int ks = slot >> 4, th = (slot >> 3) & 1, ts = (slot & 7) >> 1, eo = slot & 1;
      const int g = lane & 7, wsel = lane >> 3;  // wsel = mt >> 2
      const float* sr = Y + (size_t)(2 * EB + e) * Cfg::FP;  // S r_v of this entry
      unsigned own = 0u, bits = 0u;
#pragma unroll
      for (int mq = 0; mq < 4; ++mq)
#pragma unroll
        for (int rh = 0; rh < 2; ++rh) {
          const int mt = 4 * wsel + mq;
          const unsigned pos = 16u * eo + 4u * mq + 2u * rh + th;
          own |= 1u << pos;
          bits |= (sr[16 * mt + 8 * rh + g] >= 0.f ? 1u : 0u) << pos;
        }
      unsigned* wp = reinterpret_cast<unsigned*>(vt + Vs::kOffVS + word_offset(Vs::KSW, ks * (D / 64) + wsel, 4 * g + ts));
      *wp = (__ldcg(wp) & ~own) | bits;
      if (lane == 0) reinterpret_cast<unsigned short*>(vt + Vs::kOffVR)[slot_lane(slot)] = f32_to_f16_bits_clamped(nrm[3][e]);
    }
  }
  if (lane < EPW) {
    const int e = warp + lane * NW;
    if (e < nb && !s_full[e]) {
      int slot;
      unsigned char* tp = tile_of(e, slot);
      const int nl = slot_lane(slot);
      const unsigned short rn = a.literal ? literal_rnorm_bits(__ldg(a.ebar_k + lh), D) : f32_to_f16_bits_clamped(nrm[1][e]);
      reinterpret_cast<unsigned*>(tp + Lo::kOffNK)[nl] = (unsigned)f32_to_f16_bits_clamped(nrm[0][e]) | ((unsigned)rn << 16);
      reinterpret_cast<unsigned short*>(tp + Lo::kOffVN)[nl] = f32_to_f16_bits_clamped(nrm[2][e]);
    }
  }
  // ---- arrival: the last head of a batch entry publishes the new length
  __syncthreads();
  if (tid < nb) {
    const int lb = layer * B + b0 + tid;
    __threadfence();
    const int old = atomicAdd(&a.cv.arrive[lb], 1);
    if (old == H - 1) {
      a.cv.arrive[lb] = 0;
      if (s_full[tid]) atomicExch(a.cv.status, (int)TQ_ERR_CAPACITY);
      else a.cv.seq_len[lb] = s_len0[tid] + 1;
      __threadfence();
    }
  }
}

template <int D, typename T, int EB>
static cudaError_t launch_prep_e(const PrepArgs& a, int lh_count, int B, bool do_append, bool do_query, cudaStream_t st) {
  using Cfg = PrepCfg<D, EB>;
  const int grid = lh_count * ((B + EB - 1) / EB);
  const int smem = (int)Cfg::kSmemBytes;
  cudaError_t e;
  // the attribute is set per launch: it is per device and a process may drive several
  if (do_append && do_query) {
    if ((e = cudaFuncSetAttribute(prep_kernel<D, T, true, true, EB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    prep_kernel<D, T, true, true, EB><<<grid, kPrepThreads, smem, st>>>(a);
  } else if (do_append) {
    if ((e = cudaFuncSetAttribute(prep_kernel<D, T, true, false, EB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    prep_kernel<D, T, true, false, EB><<<grid, kPrepThreads, smem, st>>>(a);
  } else {
    if ((e = cudaFuncSetAttribute(prep_kernel<D, T, false, true, EB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    prep_kernel<D, T, false, true, EB><<<grid, kPrepThreads, smem, st>>>(a);
  }
  count_launch();
  return cudaGetLastError();
}

template <int D, typename T>
static cudaError_t launch_prep_t(const PrepArgs& a, int lh_count, int B, int num_sms, bool do_append, bool do_query, cudaStream_t st) {
  // 32 entries per CTA when that still gives every SM a few CTAs (fewest instructions per unit), else 8 (shortest CTA)
  if ((long)lh_count * ((B + 31) / 32) >= 2L * num_sms) return launch_prep_e<D, T, 32>(a, lh_count, B, do_append, do_query, st);
  return launch_prep_e<D, T, 8>(a, lh_count, B, do_append, do_query, st);
}

cudaError_t launch_prep(const DecodeArgs& d, const void* k, const void* v, int D, int num_sms, bool do_append,
                        bool do_query, cudaStream_t st) {
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
  a.frags = d.frags;
  a.tabs = d.tabs;
  a.layer_begin = d.layer_begin;
  a.rope_layout = d.rope_layout;
  a.literal = d.literal;
  a.ebar_k = d.ebar_k;
  const int lh_count = d.n_layers_call * d.cv.H;
  if (D == 64)
    return d.dt == TQ_F16 ? launch_prep_t<64, __half>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st)
                          : launch_prep_t<64, float>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st);
  return d.dt == TQ_F16 ? launch_prep_t<128, __half>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st)
                        : launch_prep_t<128, float>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st);
}

}  // namespace tq
