// tq_quantize_tc.cu — KV quantize-and-pack on the 5th-generation tensor cores (tcgen05 + TMEM), head_dim 64 and 128.
//
// Same arithmetic as tq_quantize.cu (PAPER.md:111-116 prefill steps 1,3,4; §3.3 Eq. 5; §3.4 Eq. 6 in the sign(S r)
// form of BASELINE.json:north_star), but the three rotations y = PI_K x', S r, PI_V v — a dense
// (tokens x d) x (d x d) contraction — run as tcgen05.mma with the accumulators in tensor memory:
//   * a CTA of 128 threads owns 128-token blocks of one (batch, head): UMMA M = 128 tokens, N = d outputs, K = 16;
//     keys (RoPE, PI_K, then S on the residual) and values (PI_V) run as separate CTAs (blockIdx.z);
//   * operands are fp16 in shared memory in the canonical K-major no-swizzle layout (8 x 8 core matrices);
//     fp32 accuracy comes from two-term splits a = a_hi + a_lo (each product exact in the fp32 accumulator):
//     D = A_hi B_hi + A_lo B_hi + A_hi B_lo.  Power-of-two scalings keep every split away from the fp16 range
//     limits and cancel exactly: PI x16, the token vector by 2^-exponent(max |x|) (RoPE grows a pair by at most
//     sqrt 2), r x8 (only sign(S r) is used); fp16 values V are exact operands and need two products only.  A numpy
//     study (hard part 4) puts the code-flip rate of this scheme at 2e-7, that of an all-fp32 pipeline;
//   * the epilogue is thread-per-token: tcgen05.ld hands every thread the rotated coordinates of ITS token, 32
//     columns at a time (pass 1: the norm; pass 2: codes, residual, packing), so nothing crosses lanes.  The device
//     tile layout (tq_common.cuh) is the A-fragment order of the decode kernel's MMAs, so every thread drops its
//     bytes into an image of the block's four tiles in shared memory (byte / halfword stores; V fields, which mix the
//     two tokens of a pair, are assembled by the pair from a small per-token scratch) and the CTA then writes the
//     image out with coalesced 16-byte stores.  Tiles only partly covered by the call are pre-loaded into the image.
#include "tq_common.cuh"

namespace tq {
namespace {

constexpr int kBlk = 128;  // tokens per block = UMMA M = threads per CTA

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int D>
struct TcCfg {
  using Lo = Layout<D>;
  static constexpr int kSBO = 16 * D;              // bytes between 8-row groups of an operand: 1024 | 2048
  static constexpr int kOpBytes = kBlk * D * 2;    // one fp16 A operand: 16 | 32 KB
  static constexpr int kMatBytes = D * D * 2;      // one fp16 B operand: 8 | 32 KB
  static constexpr int kTmemCols = 2 * D;          // key CTAs: D_K [0,d), D_S [d,2d); value CTAs: D_V [0,d)
  // instruction descriptor: kind::f16, A = B = fp16 (K-major), D = fp32, N = d, M = 128
  static constexpr uint32_t kIdesc = (1u << 4) | ((uint32_t)(D >> 3) << 17) | ((128u >> 4) << 24);
  // image of one tile's sections owned by a CTA: keys [K codes | K signs | norms k,r], values [V codes | norm v]
  static constexpr int kImgK = Lo::kCodeBytes + Lo::kSignBytes + 4 * kTile;
  static constexpr int kImgV = Lo::kCodeBytes + 2 * kTile;
  static constexpr int kImgBytes = kImgK;          // per tile (the larger of the two)
  static constexpr int kScrPitch = Lo::C + 1;      // V scratch: C words (8 codes each) per token, odd pitch
  // shared memory: B operands 4 x kMatBytes (keys: PI_K hi/lo, S hi/lo; values: PI_V hi/lo) | A operands hi, lo |
  // tile images [4][kImgBytes] | V scratch [128][kScrPitch] | LUT, barriers, TMEM slot
  static constexpr int kOffA = 4 * kMatBytes, kOffMisc = kOffA + 2 * kOpBytes;
  static constexpr int kSmemBytes = kOffMisc + 4 * kImgBytes + kBlk * kScrPitch * 4 + 8 * 4 + 3 * 8 + 16;
};

// byte offset of element (row, k) of a [rows][d] fp16 operand in the canonical K-major no-swizzle layout:
// core matrix = 8 rows x 16 bytes, contiguous (128 B); K-adjacent cores 128 B apart, row-group-adjacent 16 d bytes apart
template <int D>
__device__ __forceinline__ int core_off(int row, int k) {
  return (row >> 3) * TcCfg<D>::kSBO + (k >> 3) * 128 + (row & 7) * 16 + (k & 7) * 2;
}
// shared-memory matrix descriptor of such an operand starting at byte address saddr (k-step ks adds 256 B)
template <int D>
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(TcCfg<D>::kSBO >> 4) << 32) |
         ((uint64_t)1 << 46);  // version 1 (Blackwell), no swizzle, base offset 0
}

__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred P1;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}"
      ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// 32 consecutive fp32 accumulator columns of this thread's TMEM lane (= its token)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
// two-term fp16 split of 8 consecutive values, packed as two 16-byte rows of the operand layout
__device__ __forceinline__ void split8(const float* x, uint4& hi, uint4& lo) {
  unsigned h[4], l[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {  // packed conversions: one cvt per pair each way
    const __half2 h2 = __floats2half2_rn(x[2 * j], x[2 * j + 1]);
    const float2 hf = __half22float2(h2);
    const __half2 l2 = __floats2half2_rn(x[2 * j] - hf.x, x[2 * j + 1] - hf.y);
    h[j] = *reinterpret_cast<const unsigned*>(&h2);
    l[j] = *reinterpret_cast<const unsigned*>(&l2);
  }
  hi = make_uint4(h[0], h[1], h[2], h[3]);
  lo = make_uint4(l[0], l[1], l[2], l[3]);
}

// B operand of one d x d fp32 matrix M (row-major [n][k], y = M x): hi and lo halves, scaled by `scale`
template <int D>
__device__ __forceinline__ void stage_matrix(unsigned char* bhi, unsigned char* blo, const float* __restrict__ M, float scale,
                                             int tid) {
  for (int idx = tid; idx < D * D / 8; idx += kBlk) {
    const int n = idx / (D / 8), kj = idx % (D / 8);
    const float4 a = __ldg(reinterpret_cast<const float4*>(M + n * D + 8 * kj));
    const float4 b = __ldg(reinterpret_cast<const float4*>(M + n * D + 8 * kj) + 1);
    const float x[8] = {a.x * scale, a.y * scale, a.z * scale, a.w * scale, b.x * scale, b.y * scale, b.z * scale, b.w * scale};
    uint4 hi, lo;
    split8(x, hi, lo);
    *reinterpret_cast<uint4*>(bhi + core_off<D>(n, 8 * kj)) = hi;
    *reinterpret_cast<uint4*>(blo + core_off<D>(n, 8 * kj)) = lo;
  }
}

// power-of-two scale 2^-e with 2^e <= amax < 2^(e+1) (1 for amax = 0), and its exact inverse
__device__ __forceinline__ void pow2_scale(float amax, float& s, float& inv_s) {
  unsigned E = (__float_as_uint(amax) >> 23) & 0xffu;
  E = E < 2u ? 127u : (E > 252u ? 252u : E);  // zero / denormal maxima are left unscaled
  s = __uint_as_float((254u - E) << 23);
  inv_s = __uint_as_float(E << 23);
}

// code = #{k : u > thr[k]} for ascending thresholds, as a three-step binary search (3 compares + 4 selects instead of
// 7 compares + 7 adds); identical result, ties included (u > t is evaluated on the same thresholds)
__device__ __forceinline__ int code_of(float u, const float (&thr)[7]) {
  const bool b2 = u > thr[3];
  const float tm = b2 ? thr[5] : thr[1];
  const bool b1 = u > tm;
  const float tl = b2 ? (b1 ? thr[6] : thr[4]) : (b1 ? thr[2] : thr[0]);
  const bool b0 = u > tl;
  return (b2 ? 4 : 0) + (b1 ? 2 : 0) + (b0 ? 1 : 0);
}


// 8 consecutive input values of one token as floats (zeros for a token outside the call)
template <typename T>
__device__ __forceinline__ void load8(const T* p, bool valid, float (&x)[8]) {
  if (!valid) {
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = 0.f;
    return;
  }
  if constexpr (sizeof(T) == 2) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
    const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[j]));
      x[2 * j] = f.x, x[2 * j + 1] = f.y;
    }
  } else {
    const float4 a = __ldg(reinterpret_cast<const float4*>(p)), b = __ldg(reinterpret_cast<const float4*>(p) + 1);
    x[0] = a.x, x[1] = a.y, x[2] = a.z, x[3] = a.w, x[4] = b.x, x[5] = b.y, x[6] = b.z, x[7] = b.w;
  }
}

// max |x| over one token's d input values (first pass over the row; the second pass hits L1/L2)
template <int D, typename T>
__device__ __forceinline__ float row_amax(const T* p, bool valid) {
  float amax = 0.f;
#pragma unroll 4
  for (int kj = 0; kj < D / 8; ++kj) {
    float x[8];
    load8<T>(p + 8 * kj, valid, x);
#pragma unroll
    for (int j = 0; j < 8; ++j) amax = fmaxf(amax, fabsf(x[j]));
  }
  return amax;
}

template <int D>
__device__ __forceinline__ void store_split8(const float (&x)[8], float s, unsigned char* ahi, unsigned char* alo, int row, int k0) {
  float xs[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) xs[j] = x[j] * s;
  uint4 hi, lo;
  split8(xs, hi, lo);
  *reinterpret_cast<uint4*>(ahi + core_off<D>(row, k0)) = hi;
  *reinterpret_cast<uint4*>(alo + core_off<D>(row, k0)) = lo;
}

// keys: RoPE (fp64-evaluated table), scale, split, store both operand rows; returns the exact inverse scale
template <int D, typename T>
__device__ __forceinline__ float stage_key_row(const T* p, bool valid, const float* __restrict__ cs_row /* [d/2][2] */,
                                               int rope_layout, unsigned char* ahi, unsigned char* alo, int row) {
  float s, inv_s;
  pow2_scale(row_amax<D, T>(p, valid), s, inv_s);  // |RoPE(x) s| < 2 sqrt 2
  if (rope_layout == 0) {  // pairs (2g, 2g+1): four pairs per 8-value chunk
#pragma unroll 4
    for (int kj = 0; kj < D / 8; ++kj) {
      float x[8];
      load8<T>(p + 8 * kj, valid, x);
      const float4 c0 = __ldg(reinterpret_cast<const float4*>(cs_row + 8 * kj)), c1 = __ldg(reinterpret_cast<const float4*>(cs_row + 8 * kj) + 1);
      const float cs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
      float y[8];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        y[2 * j] = x[2 * j] * cs[2 * j] - x[2 * j + 1] * cs[2 * j + 1];
        y[2 * j + 1] = x[2 * j] * cs[2 * j + 1] + x[2 * j + 1] * cs[2 * j];
      }
      store_split8<D>(y, s, ahi, alo, row, 8 * kj);
    }
  } else {  // pairs (g, g + d/2): chunk kj with chunk kj + d/16
#pragma unroll 2
    for (int kj = 0; kj < D / 16; ++kj) {
      float xa[8], xb[8], ya[8], yb[8];
      load8<T>(p + 8 * kj, valid, xa);
      load8<T>(p + D / 2 + 8 * kj, valid, xb);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float4 c = __ldg(reinterpret_cast<const float4*>(cs_row + 16 * kj) + q);  // pairs g = 8 kj + 2q, + 1
        ya[2 * q] = xa[2 * q] * c.x - xb[2 * q] * c.y, yb[2 * q] = xa[2 * q] * c.y + xb[2 * q] * c.x;
        ya[2 * q + 1] = xa[2 * q + 1] * c.z - xb[2 * q + 1] * c.w, yb[2 * q + 1] = xa[2 * q + 1] * c.w + xb[2 * q + 1] * c.z;
      }
      store_split8<D>(ya, s, ahi, alo, row, 8 * kj);
      store_split8<D>(yb, s, ahi, alo, row, D / 2 + 8 * kj);
    }
  }
  return inv_s;
}

// values: fp16 inputs are exact operands (copied as they are, no scale); fp32 inputs are scaled and split
template <int D, typename T>
__device__ __forceinline__ float stage_value_row(const T* p, bool valid, unsigned char* ahi, unsigned char* alo, int row) {
  if constexpr (sizeof(T) == 2) {
#pragma unroll 4
    for (int kj = 0; kj < D / 8; ++kj)
      *reinterpret_cast<uint4*>(ahi + core_off<D>(row, 8 * kj)) =
          valid ? __ldg(reinterpret_cast<const uint4*>(p) + kj) : make_uint4(0, 0, 0, 0);
    return 1.f;
  } else {
    float s, inv_s;
    pow2_scale(row_amax<D, T>(p, valid), s, inv_s);
#pragma unroll 4
    for (int kj = 0; kj < D / 8; ++kj) {
      float x[8];
      load8<T>(p + 8 * kj, valid, x);
      store_split8<D>(x, s, ahi, alo, row, 8 * kj);
    }
    return inv_s;
  }
}

template <int D, typename T, bool kKey>
__device__ __forceinline__ void quantize_pack_tc_body(const QuantArgs& a, int blocks_per_cta, unsigned char* smem) {
  using Cfg = TcCfg<D>;
  using Lo = Layout<D>;
  constexpr bool kF16 = sizeof(T) == 2;
  constexpr int KCW = Lo::KCW, KSW = Lo::KSW, P = Lo::P;
  unsigned char *B0_hi = smem, *B0_lo = smem + Cfg::kMatBytes;                               // PI_K | PI_V
  unsigned char *B1_hi = smem + 2 * Cfg::kMatBytes, *B1_lo = smem + 3 * Cfg::kMatBytes;      // S (keys only)
  unsigned char *A_hi = smem + Cfg::kOffA, *A_lo = A_hi + Cfg::kOpBytes;
  unsigned char* img = smem + Cfg::kOffMisc;                                  // [4 tiles][kImgBytes]
  unsigned* vscr = reinterpret_cast<unsigned*>(img + 4 * Cfg::kImgBytes);     // [128][kScrPitch] V code groups
  float* lut_s = reinterpret_cast<float*>(vscr + kBlk * Cfg::kScrPitch);      // [8]
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(lut_s + 8);  // [0]: first product, [1]: S product
  unsigned* tmem_slot = reinterpret_cast<unsigned*>(mbar + 3);

  const int tid = threadIdx.x, warp = tid >> 5;
  const int bh = blockIdx.y, b = bh / a.cv.H, h = bh % a.cv.H;
  const int first_blk = a.start_pos / kBlk, last_blk = (a.start_pos + a.n_tokens - 1) / kBlk;
  const int blk0 = first_blk + (int)blockIdx.x * blocks_per_cta;
  if (blk0 > last_blk) return;
  const int blk1 = min(last_blk, blk0 + blocks_per_cta - 1);
  if (kKey && blockIdx.x == 0 && h == 0 && tid == 0) a.cv.seq_len[a.layer * a.cv.B + b] = a.start_pos + a.n_tokens;

  // ---- one-time setup: tensor memory, barriers, the B operands of this head, LUT
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                 "r"(Cfg::kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 0) {
    mbar_init(smem_u32(mbar + 0), 1);
    mbar_init(smem_u32(mbar + 1), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if constexpr (kKey) {
    stage_matrix<D>(B0_hi, B0_lo, a.pi_k + (size_t)h * D * D, 16.f, tid);
    stage_matrix<D>(B1_hi, B1_lo, a.S, 1.f, tid);
  } else {
    stage_matrix<D>(B0_hi, B0_lo, a.pi_v + (size_t)h * D * D, 16.f, tid);
  }
  float thr[7];
  {
    const float* lut_g = (kKey ? a.lut_k : a.lut_v) + h * 8;
    float l8[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) l8[q] = __ldg(lut_g + q);
#pragma unroll
    for (int q = 0; q < 7; ++q) thr[q] = 0.5f * (l8[q] + l8[q + 1]);
    if (tid < 8) lut_s[tid] = __ldg(lut_g + tid);
  }
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);  // this warp's quadrant of TMEM lanes
  const uint32_t a_hi = smem_u32(A_hi), a_lo = smem_u32(A_lo), b0_hi = smem_u32(B0_hi), b0_lo = smem_u32(B0_lo),
                 b1_hi = smem_u32(B1_hi), b1_lo = smem_u32(B1_lo);
  auto gemm = [&](uint32_t dcol, uint32_t a_op, uint32_t b_op, bool first) {  // D[:, dcol..dcol+d) (+)= A B^T, K = d
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks)
      umma_f16(tmem + dcol, umma_desc<D>(a_op + ks * 256), umma_desc<D>(b_op + ks * 256), Cfg::kIdesc,
               (first && ks == 0) ? 0u : 1u);
  };

  const T* src = reinterpret_cast<const T*>(kKey ? a.k : a.v) + (size_t)bh * a.n_tokens * D;
  unsigned char* stream = a.cv.tiles + ((size_t)a.layer * a.cv.B * a.cv.H + bh) * a.cv.stream_bytes;
  const int slot = tid & 31, tl = tid >> 5, sg = slot & 7, sr = slot >> 3;
  unsigned char* timg = img + tl * Cfg::kImgBytes;  // image of this token's tile
  constexpr int kOffImgKS = Lo::kCodeBytes, kOffImgNK = Lo::kCodeBytes + Lo::kSignBytes;  // keys image
  constexpr int kOffImgVN = Lo::kCodeBytes;                                                // values image
  // byte `sb` of lane l's word string in a section of W words per lane
  auto sec_byte = [](int W, int l, int sb) { return word_offset(W, sb >> 2, l) + (sb & 3); };

  for (int blk = blk0; blk <= blk1; ++blk) {
    const uint32_t parity = (uint32_t)(blk - blk0) & 1u;
    const int pos = blk * kBlk + tid;
    const int i = pos - a.start_pos;
    const bool valid = i >= 0 && i < a.n_tokens;
    // tiles of this block: covered (some token of the call) / fully covered; partly covered ones are pre-loaded so that
    // the bits of tokens outside the call survive the write-back
    const int call_end = a.start_pos + a.n_tokens;
    auto tile_cover = [&](int t4) {  // 0 none, 1 partial, 2 full
      const int p0 = blk * kBlk + t4 * kTile, lo = max(p0, a.start_pos), hi = min(p0 + kTile, call_end);
      return hi <= lo ? 0 : (hi - lo == kTile ? 2 : 1);
    };
    {
      constexpr int kOwn = kKey ? Cfg::kImgK : Cfg::kImgV;
      for (int idx = tid; idx < 4 * (kOwn / 16); idx += kBlk) {
        const int t4 = idx / (kOwn / 16), q = idx % (kOwn / 16);
        if (tile_cover(t4) != 1) continue;
        const unsigned char* tg = stream + (size_t)(blk * 4 + t4) * Lo::kTileBytes;
        // keys: [0, kOffVC) then the norms; values: the V codes then |v|
        const int ib = 16 * q;
        const int gb = kKey ? (ib < Lo::kOffVC ? ib : Lo::kOffNK + (ib - Lo::kOffVC))
                            : (ib < Lo::kCodeBytes ? Lo::kOffVC + ib : Lo::kOffVN + (ib - Lo::kCodeBytes));
        *reinterpret_cast<uint4*>(img + t4 * Cfg::kImgBytes + ib) = *reinterpret_cast<const uint4*>(tg + gb);
      }
    }

    // ---- stage the A operand rows of this thread's token and start the first product
    float inv_s;
    if constexpr (kKey)
      inv_s = stage_key_row<D, T>(src + (size_t)i * D, valid, a.rope_cs + (size_t)min(pos, a.cv.max_seq - 1) * D, a.rope_layout,
                                  A_hi, A_lo, tid);
    else
      inv_s = stage_value_row<D, T>(src + (size_t)i * D, valid, A_hi, A_lo, tid);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
      gemm(0, a_hi, b0_hi, true), gemm(0, a_hi, b0_lo, false);
      if (kKey || !kF16) gemm(0, a_lo, b0_hi, false);
      umma_commit(smem_u32(mbar + 0));
    }
    mbar_wait(smem_u32(mbar + 0), parity);
    tc_fence_after();

    // ---- thread = token, pass 1: |y|^2 over the d accumulator columns
    float n2 = 0.f;
#pragma unroll 1
    for (int c = 0; c < D / 32; ++c) {
      float y[32];
      tmem_ld32(t_lane + 32 * c, y);
#pragma unroll
      for (int j = 0; j < 32; ++j) n2 = fmaf(y[j], y[j], n2);
    }
    const float n = sqrtf(n2);
    const float inv = n > 0.f ? 1.0f / n : 0.f;
    const unsigned short n_h = f32_to_f16_bits_clamped(n * inv_s * 0.0625f);  // y = 16 s PI x

    if constexpr (kKey) {
      // ---- pass 2: codes, residual (the A operand of the S product); the pair fields go straight into the tile image:
      //      pair p = 16 c + g belongs to lane (sg, t = g & 3) as field j = 4 c + (g >> 2) of this token's block
      //      (bits [6 J sr + 6 j, + 6) of the lane's string): four fields = three bytes per lane and chunk
      float g2 = 0.f;
#pragma unroll 1
      for (int c = 0; c < D / 32; ++c) {
        float y[32];
        tmem_ld32(t_lane + 32 * c, y);
        unsigned yt[4] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int g = 0; g < 16; ++g) {
          const float u0 = y[2 * g] * inv, u1 = y[2 * g + 1] * inv;
          const int c0 = code_of(u0, thr), c1 = code_of(u1, thr);
          const float r0 = u0 - lut_s[c0], r1 = u1 - lut_s[c1];
          g2 = fmaf(r0, r0, fmaf(r1, r1, g2));
          y[2 * g] = r0 * 8.f, y[2 * g + 1] = r1 * 8.f;  // scaled for the fp16 split (only sign(S r) is used)
          yt[g & 3] |= (unsigned)(c0 | (c1 << 3)) << (6 * (g >> 2));
        }
        if (valid) {
#pragma unroll
          for (int t = 0; t < 4; ++t) {
            const int sb = (6 * Lo::J * sr) / 8 + 3 * c;  // byte of the lane's K string
#pragma unroll
            for (int k = 0; k < 3; ++k) timg[sec_byte(KCW, 4 * sg + t, sb + k)] = (unsigned char)(yt[t] >> (8 * k));
          }
        }
#pragma unroll
        for (int kj = 0; kj < 4; ++kj) {  // the first product is complete (barrier): the A buffers are free
          uint4 hi, lo;
          split8(&y[8 * kj], hi, lo);
          *reinterpret_cast<uint4*>(A_hi + core_off<D>(tid, 32 * c + 8 * kj)) = hi;
          *reinterpret_cast<uint4*>(A_lo + core_off<D>(tid, 32 * c + 8 * kj)) = lo;
        }
      }
      fence_async_smem();
      tc_fence_before();
      __syncthreads();
      if (tid == 0) {
        tc_fence_after();
        gemm(D, a_hi, b1_hi, true), gemm(D, a_lo, b1_hi, false), gemm(D, a_hi, b1_lo, false);
        umma_commit(smem_u32(mbar + 1));
      }
      if (valid)
        reinterpret_cast<unsigned*>(timg + kOffImgNK)[slot_lane(slot)] =
            (unsigned)n_h | ((unsigned)f32_to_f16_bits_clamped(sqrtf(g2)) << 16);
      // ---- residual sketch: bit j = [(S r)_j >= 0].  Sketch rows [t d/4, (t+1) d/4) belong to lane (sg, t) as 16-bit
      //      pieces u; a piece is stored as two bytes of word (mt, u): byte (sr & 1) holds bits 0..7, byte 2 + (sr & 1)
      //      bits 8..15 (the byte interleave with the slot 8 further on makes the decode kernel's fp16x2 masks work)
      mbar_wait(smem_u32(mbar + 1), parity);
      tc_fence_after();
#pragma unroll 1
      for (int c = 0; c < D / 32; ++c) {
        float y[32];
        tmem_ld32(t_lane + D + 32 * c, y);
        unsigned w = 0u;
#pragma unroll
        for (int j = 0; j < 32; ++j) w |= (y[j] >= 0.f ? 1u : 0u) << j;
        if (valid) {
#pragma unroll
          for (int q = 0; q < 2; ++q) {
            const int rho0 = 32 * c + 16 * q, t = rho0 / (D / 4), u = (rho0 % (D / 4)) >> 4;
            const int word = (sr >> 1) * Lo::U + u;
            unsigned char* wp = timg + kOffImgKS + word_offset(KSW, word, 4 * sg + t);
            wp[sr & 1] = (unsigned char)(w >> (16 * q));
            wp[2 + (sr & 1)] = (unsigned char)(w >> (16 * q + 8));
          }
        }
      }
    } else {
      // ---- values, pass 2: codes, eight per scratch word; then the two tokens of a pair assemble the six-bit fields
      //      code_i(even token) | code_i(odd token) << 3 of lane (i & 7, pp & 3), block j = pp >> 2: the even token
      //      builds the lanes i & 7 < 4, the odd one the others
      unsigned* myg = vscr + tid * Cfg::kScrPitch;
#pragma unroll 1
      for (int c = 0; c < D / 32; ++c) {
        float y[32];
        tmem_ld32(t_lane + 32 * c, y);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          unsigned w = 0;
#pragma unroll
          for (int i = 0; i < 8; ++i) w |= (unsigned)code_of(y[8 * q + i] * inv, thr) << (3 * i);
          myg[4 * c + q] = w;
        }
      }
      if (valid) reinterpret_cast<unsigned short*>(timg + kOffImgVN)[slot_lane(slot)] = n_h;
      __syncwarp();
      {
        const int e = slot & 1, pp = slot >> 1;
        const unsigned* ge = vscr + (tid & ~1) * Cfg::kScrPitch;  // even token of the pair
        const unsigned* go = ge + Cfg::kScrPitch;                 // odd token
        const bool v_e = __shfl_sync(0xffffffffu, valid, (slot & ~1)), v_o = __shfl_sync(0xffffffffu, valid, (slot | 1));
        if (v_e || v_o) {
          constexpr int HW = 3 * D / 64;  // halfwords per (lane, token pair) block
#pragma unroll
          for (int gq = 0; gq < 4; ++gq) {
            const int gi = 4 * e + gq;
            unsigned short hw16[HW];
#pragma unroll
            for (int h = 0; h < HW; ++h) hw16[h] = 0;
            unsigned long long acc = 0ull;  // fields stream through a 64-bit window, 16 bits out at a time
            int nbits = 0, hout = 0;
#pragma unroll
            for (int c = 0; c < Lo::C; ++c) {
              const unsigned f = ((ge[c] >> (3 * gi)) & 7u) | (((go[c] >> (3 * gi)) & 7u) << 3);
              acc |= (unsigned long long)f << nbits;
              nbits += 6;
              if (nbits >= 16) {
                hw16[hout++] = (unsigned short)acc;
                acc >>= 16, nbits -= 16;
              }
            }
            const unsigned short keep_mask = (v_e && v_o) ? 0u : 0xffffu;  // partial pair: read-modify-write
#pragma unroll
            for (int h = 0; h < HW; ++h) {
              const int hidx = (pp >> 2) * HW + h;
              unsigned short* dst =
                  reinterpret_cast<unsigned short*>(timg + word_offset(KCW, hidx >> 1, 4 * gi + (pp & 3))) + (hidx & 1);
              if (keep_mask) {
                // bits of the valid token inside this halfword: three of every six, phase by the bit offset 16 h
                unsigned short m = 0;
#pragma unroll
                for (int bit = 0; bit < 16; ++bit) {
                  const int fb = (16 * h + bit) % 6;
                  if ((fb < 3) == v_e) m |= (unsigned short)(1u << bit);
                }
                *dst = (unsigned short)((*dst & ~m) | (hw16[h] & m));
              } else {
                *dst = hw16[h];
              }
            }
          }
        }
      }
    }
    // ---- write the block's tile images out (every tile the call touches; the image of a partly covered tile carries
    //      the old bits of the other tokens)
    __syncthreads();
    {
      constexpr int kOwn = kKey ? Cfg::kImgK : Cfg::kImgV;
      for (int idx = tid; idx < 4 * (kOwn / 16); idx += kBlk) {
        const int t4 = idx / (kOwn / 16), q = idx % (kOwn / 16);
        if (tile_cover(t4) == 0) continue;
        unsigned char* tg = stream + (size_t)(blk * 4 + t4) * Lo::kTileBytes;
        const int ib = 16 * q;
        const int gb = kKey ? (ib < Lo::kOffVC ? ib : Lo::kOffNK + (ib - Lo::kOffVC))
                            : (ib < Lo::kCodeBytes ? Lo::kOffVC + ib : Lo::kOffVN + (ib - Lo::kCodeBytes));
        *reinterpret_cast<uint4*>(tg + gb) = *reinterpret_cast<const uint4*>(img + t4 * Cfg::kImgBytes + ib);
      }
    }
    __syncthreads();  // the next block pre-loads into / writes the same images
    tc_fence_before();  // the next block's MMAs overwrite the accumulators every thread has just read
  }
  __syncthreads();
  if (warp == 0) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(Cfg::kTmemCols) : "memory");
  }
}

template <int D, typename T>
__global__ void __launch_bounds__(kBlk) quantize_pack_tc_kernel(QuantArgs a, int blocks_per_cta) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  if (blockIdx.z == 0) quantize_pack_tc_body<D, T, true>(a, blocks_per_cta, smem_dyn);
  else quantize_pack_tc_body<D, T, false>(a, blocks_per_cta, smem_dyn);
}

template <int D, typename T>
cudaError_t launch_quant_tc_t(const QuantArgs& a, int num_sms, cudaStream_t st) {
  const size_t smem = TcCfg<D>::kSmemBytes;
  const int first_blk = a.start_pos / kBlk, last_blk = (a.start_pos + a.n_tokens - 1) / kBlk;
  const int nblk = last_blk - first_blk + 1;
  const int BH = a.cv.B * a.cv.H;
  const long want = 4L * num_sms;  // CTAs per operand: enough to balance the SMs, few enough to amortise the matrices
  int bpc = (int)(((long)nblk * BH + want - 1) / want);
  bpc = bpc < 1 ? 1 : (bpc > 16 ? 16 : bpc);
  dim3 grid((nblk + bpc - 1) / bpc, BH, 2);  // z: keys | values
  cudaError_t e = cudaFuncSetAttribute(quantize_pack_tc_kernel<D, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  quantize_pack_tc_kernel<D, T><<<grid, kBlk, smem, st>>>(a, bpc);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_quantize_pack_tc(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st) {
  if (D == 64) return dt == TQ_F16 ? launch_quant_tc_t<64, __half>(a, num_sms, st) : launch_quant_tc_t<64, float>(a, num_sms, st);
  return dt == TQ_F16 ? launch_quant_tc_t<128, __half>(a, num_sms, st) : launch_quant_tc_t<128, float>(a, num_sms, st);
}

}  // namespace tq
