// tq_quantize_tc.cu — KV quantize-and-pack for head_dim 64 on the 5th-generation tensor cores (tcgen05 + TMEM).
//
// Same arithmetic as tq_quantize.cu (PAPER.md:111-116 prefill steps 1,3,4; §3.3 Eq. 5; §3.4 Eq. 6 in the sign(S r)
// form of BASELINE.json:north_star), but the three rotations y = PI_K x', S r, PI_V v — a dense
// (tokens x 64) x (64 x 64) contraction — run as tcgen05.mma with the accumulators in tensor memory:
//   * a CTA of 128 threads owns 128-token blocks of one (batch, head): UMMA M = 128 tokens, N = 64 outputs, K = 16;
//   * operands are fp16 in shared memory in the canonical K-major no-swizzle layout (8 x 8 core matrices);
//     fp32 accuracy comes from two-term splits a = a_hi + a_lo (each product exact in the fp32 accumulator):
//     D = A_hi B_hi + A_lo B_hi + A_hi B_lo.  Power-of-two scalings keep every split away from the fp16 range
//     limits and cancel exactly: PI x16, x' by 2^-exponent(max |x'|) per token, r x8 (only sign(S r) is used);
//     fp16 values V are exact operands and need two products only.  A numpy study (hard part 4)
//     puts the code-flip rate of this scheme at 2e-7, the same as an all-fp32 pipeline;
//   * the epilogue is thread-per-token: tcgen05.ld hands every thread the 64 rotated coordinates of ITS token, so
//     the norm, the codes, the residual and the bit packing need no cross-lane traffic at all, and lane = token is
//     exactly the order of the device tile layout (coalesced 16-byte stores).  Only the V codes, which the cache
//     stores per coordinate pair across tokens, go through a shared-memory transpose.
#include "tq_common.cuh"

namespace tq {
namespace {

constexpr int kD = 64;
constexpr int kBlk = 128;             // tokens per block = UMMA M = threads per CTA
constexpr int kOpBytes = kBlk * kD * 2;  // one fp16 A operand: 16 KB
constexpr int kMatBytes = kD * kD * 2;   // one fp16 B operand: 8 KB
constexpr int kTmemCols = 128;        // key CTAs: D_K [0,64), D_S [64,128); value CTAs: D_V [0,64)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// byte offset of element (row, k) of a [rows][64] fp16 operand in the canonical K-major no-swizzle layout:
// core matrix = 8 rows x 16 bytes, contiguous (128 B); K-adjacent cores 128 B apart, row-group-adjacent 1024 B apart
__device__ __forceinline__ int core_off(int row, int k) {
  return (row >> 3) * 1024 + (k >> 3) * 128 + (row & 7) * 16 + (k & 7) * 2;
}
// shared-memory matrix descriptor of such an operand starting at byte address saddr (k-step ks adds 256 B)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46);  // version 1 (Blackwell), no swizzle, base offset 0
}
// instruction descriptor: kind::f16, A = B = fp16 (K-major), D = fp32, N = 64, M = 128
constexpr uint32_t kIdesc = (1u << 4) | ((64u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(kIdesc), "r"(accumulate)
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
__device__ __forceinline__ void tmem_ld64(uint32_t taddr, float (&v)[64]) {
  float a[32], b[32];
  tmem_ld32(taddr, a);
  tmem_ld32(taddr + 32, b);
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = a[i], v[32 + i] = b[i];
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

// B operand of one 64 x 64 fp32 matrix M (row-major [n][k], y = M x): hi and lo halves, scaled by `scale`
__device__ __forceinline__ void stage_matrix(unsigned char* bhi, unsigned char* blo, const float* __restrict__ M, float scale,
                                             int tid) {
  for (int idx = tid; idx < kD * kD / 8; idx += kBlk) {
    const int n = idx >> 3, kj = idx & 7;
    const float4 a = __ldg(reinterpret_cast<const float4*>(M + n * kD + 8 * kj));
    const float4 b = __ldg(reinterpret_cast<const float4*>(M + n * kD + 8 * kj) + 1);
    const float x[8] = {a.x * scale, a.y * scale, a.z * scale, a.w * scale, b.x * scale, b.y * scale, b.z * scale, b.w * scale};
    uint4 hi, lo;
    split8(x, hi, lo);
    *reinterpret_cast<uint4*>(bhi + core_off(n, 8 * kj)) = hi;
    *reinterpret_cast<uint4*>(blo + core_off(n, 8 * kj)) = lo;
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

template <typename T>
__device__ __forceinline__ void load_vec64(const T* p, float (&x)[64]);
template <>
__device__ __forceinline__ void load_vec64<__half>(const __half* p, float (&x)[64]) {
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(p) + c);
    const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w[j]));
      x[8 * c + 2 * j] = f.x;
      x[8 * c + 2 * j + 1] = f.y;
    }
  }
}
template <>
__device__ __forceinline__ void load_vec64<float>(const float* p, float (&x)[64]) {
#pragma unroll
  for (int c = 0; c < 16; ++c) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(p) + c);
    x[4 * c] = v.x, x[4 * c + 1] = v.y, x[4 * c + 2] = v.z, x[4 * c + 3] = v.w;
  }
}

// scale a token vector into (-2, 2), split it and write both operand rows; returns the exact inverse scale
__device__ __forceinline__ float stage_split(const float (&x)[64], unsigned char* ahi, unsigned char* alo, int row) {
  float amax = 0.f;
#pragma unroll
  for (int i = 0; i < 64; ++i) amax = fmaxf(amax, fabsf(x[i]));
  float s, inv_s;
  pow2_scale(amax, s, inv_s);
#pragma unroll
  for (int kj = 0; kj < 8; ++kj) {
    float xs[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) xs[j] = x[8 * kj + j] * s;
    uint4 hi, lo;
    split8(xs, hi, lo);
    *reinterpret_cast<uint4*>(ahi + core_off(row, 8 * kj)) = hi;
    *reinterpret_cast<uint4*>(alo + core_off(row, 8 * kj)) = lo;
  }
  return inv_s;
}

// Shared memory of one CTA (keys and values run as separate CTAs, blockIdx.z, so that three of them fit an SM):
//   B operands 4 x 8 KB (keys: PI_K hi/lo, S hi/lo; values: PI_V hi/lo) | A operands 2 x 16 KB (hi, lo) | staging, LUT,
//   barriers
constexpr int kOffA = 4 * kMatBytes, kOffMisc = kOffA + 2 * kOpBytes;
constexpr int kSmemBytes = kOffMisc + kBlk * 32 + kBlk * 7 * 4 + 8 * 4 + 3 * 8 + 16;

template <typename T, bool kKey>
__device__ __forceinline__ void quantize_pack_tc_body(const QuantArgs& a, int blocks_per_cta, unsigned char* smem) {
  using Lo = Layout<kD>;
  constexpr bool kF16 = sizeof(T) == 2;
  unsigned char *Bk_hi = smem, *Bk_lo = smem + kMatBytes, *Bs_hi = smem + 2 * kMatBytes, *Bs_lo = smem + 3 * kMatBytes,
                *Bv_hi = smem, *Bv_lo = smem + kMatBytes;
  unsigned char *A_hi = smem + kOffA, *A_lo = A_hi + kOpBytes, *AV_hi = A_hi, *AV_lo = A_lo;
  unsigned char* cbV = smem + kOffMisc;                                  // [128 tokens][32 pair fields]
  unsigned* crot = reinterpret_cast<unsigned*>(cbV + kBlk * 32);          // [128][7] K code words, rotation staging
  float* lutK = reinterpret_cast<float*>(crot + kBlk * 7);                // [8]
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(lutK + 8);  // [3]: K, V, S accumulators ready
  unsigned* tmem_slot = reinterpret_cast<unsigned*>(mbar + 3);

  const int tid = threadIdx.x, warp = tid >> 5;
  const int bh = blockIdx.y, b = bh / a.cv.H, h = bh % a.cv.H;
  const int first_blk = a.start_pos / kBlk, last_blk = (a.start_pos + a.n_tokens - 1) / kBlk;
  const int blk0 = first_blk + (int)blockIdx.x * blocks_per_cta;
  if (blk0 > last_blk) return;
  const int blk1 = min(last_blk, blk0 + blocks_per_cta - 1);
  if (kKey && blockIdx.x == 0 && h == 0 && tid == 0) a.cv.seq_len[a.layer * a.cv.B + b] = a.start_pos + a.n_tokens;

  // ---- one-time setup: tensor memory, barriers, the three B operands of this head, LUTs
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(kTmemCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 0) {
    mbar_init(smem_u32(mbar + 0), 1);
    mbar_init(smem_u32(mbar + 1), 1);
    mbar_init(smem_u32(mbar + 2), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if constexpr (kKey) {
    stage_matrix(Bk_hi, Bk_lo, a.pi_k + (size_t)h * kD * kD, 16.f, tid);
    stage_matrix(Bs_hi, Bs_lo, a.S, 1.f, tid);
  } else {
    stage_matrix(Bv_hi, Bv_lo, a.pi_v + (size_t)h * kD * kD, 16.f, tid);
  }
  float thrK[7], thrV[7], lutVr[8];
  {
    float lk[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) lk[q] = __ldg(a.lut_k + h * 8 + q), lutVr[q] = __ldg(a.lut_v + h * 8 + q);
#pragma unroll
    for (int q = 0; q < 7; ++q) thrK[q] = 0.5f * (lk[q] + lk[q + 1]), thrV[q] = 0.5f * (lutVr[q] + lutVr[q + 1]);
    if (tid < 8) lutK[tid] = lk[tid & 7];
  }
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t t_lane = tmem + ((uint32_t)(warp * 32) << 16);  // this warp's quadrant of TMEM lanes
  const uint32_t aK_hi = smem_u32(A_hi), aK_lo = smem_u32(A_lo), aV_hi = smem_u32(AV_hi), aV_lo = smem_u32(AV_lo);
  const uint32_t bK_hi = smem_u32(Bk_hi), bK_lo = smem_u32(Bk_lo), bS_hi = smem_u32(Bs_hi), bS_lo = smem_u32(Bs_lo),
                 bV_hi = smem_u32(Bv_hi), bV_lo = smem_u32(Bv_lo);
  auto gemm = [&](uint32_t dcol, uint32_t a_op, uint32_t b_op, bool first) {  // D[:, dcol..dcol+64) (+)= A B^T, K = 64
#pragma unroll
    for (int ks = 0; ks < kD / 16; ++ks)
      umma_f16(tmem + dcol, umma_desc(a_op + ks * 256), umma_desc(b_op + ks * 256), (first && ks == 0) ? 0u : 1u);
  };

  const T* ksrc = reinterpret_cast<const T*>(a.k) + (size_t)bh * a.n_tokens * kD;
  const T* vsrc = reinterpret_cast<const T*>(a.v) + (size_t)bh * a.n_tokens * kD;
  unsigned char* stream = a.cv.tiles + ((size_t)a.layer * a.cv.B * a.cv.H + bh) * a.cv.stream_bytes;
  const int slot = tid & 31;

  for (int blk = blk0; blk <= blk1; ++blk) {
    const uint32_t parity = (uint32_t)(blk - blk0) & 1u;
    const int pos = blk * kBlk + tid;
    const int i = pos - a.start_pos;
    const bool valid = i >= 0 && i < a.n_tokens;
    unsigned char* tp = stream + (size_t)(pos / kTile) * Lo::kTileBytes;

    // ---- stage the A operands: RoPE'd, scaled, split keys; values (exact fp16 operands when the input is fp16)
    float inv_sk = 1.f, inv_sv = 1.f;
    if constexpr (kKey) {
      float x[64];
      if (valid) load_vec64<T>(ksrc + (size_t)i * kD, x);
      else {
#pragma unroll
        for (int j = 0; j < 64; ++j) x[j] = 0.f;
      }
      const float4* cs4 = reinterpret_cast<const float4*>(a.rope_cs + (size_t)min(pos, a.cv.max_seq - 1) * kD);
#pragma unroll
      for (int g2 = 0; g2 < 16; ++g2) {  // two rotation pairs per 16-byte table read
        const float4 cs = __ldg(cs4 + g2);
        if (a.rope_layout == 0) {
          const float a0 = x[4 * g2], b0 = x[4 * g2 + 1], a1 = x[4 * g2 + 2], b1 = x[4 * g2 + 3];
          x[4 * g2] = a0 * cs.x - b0 * cs.y, x[4 * g2 + 1] = a0 * cs.y + b0 * cs.x;
          x[4 * g2 + 2] = a1 * cs.z - b1 * cs.w, x[4 * g2 + 3] = a1 * cs.w + b1 * cs.z;
        } else {
          const float a0 = x[2 * g2], b0 = x[2 * g2 + 32], a1 = x[2 * g2 + 1], b1 = x[2 * g2 + 33];
          x[2 * g2] = a0 * cs.x - b0 * cs.y, x[2 * g2 + 32] = a0 * cs.y + b0 * cs.x;
          x[2 * g2 + 1] = a1 * cs.z - b1 * cs.w, x[2 * g2 + 33] = a1 * cs.w + b1 * cs.z;
        }
      }
      inv_sk = stage_split(x, A_hi, A_lo, tid);
    } else if (kF16) {
#pragma unroll
      for (int kj = 0; kj < 8; ++kj) {
        const uint4 v = valid ? __ldg(reinterpret_cast<const uint4*>(vsrc + (size_t)i * kD) + kj) : make_uint4(0, 0, 0, 0);
        *reinterpret_cast<uint4*>(AV_hi + core_off(tid, 8 * kj)) = v;
      }
    } else {
      float x[64];
      if (valid) load_vec64<T>(vsrc + (size_t)i * kD, x);
      else {
#pragma unroll
        for (int j = 0; j < 64; ++j) x[j] = 0.f;
      }
      inv_sv = stage_split(x, AV_hi, AV_lo, tid);
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
      if constexpr (kKey) {
        gemm(0, aK_hi, bK_hi, true), gemm(0, aK_lo, bK_hi, false), gemm(0, aK_hi, bK_lo, false);
        umma_commit(smem_u32(mbar + 0));
      } else {
        gemm(0, aV_hi, bV_hi, true), gemm(0, aV_hi, bV_lo, false);
        if (!kF16) gemm(0, aV_lo, bV_hi, false);
        umma_commit(smem_u32(mbar + 1));
      }
    }

    // ---- keys: thread = token.  y = D_K / (16 s): norm, unit vector, codes, residual, its norm
    if constexpr (kKey) {
    mbar_wait(smem_u32(mbar + 0), parity);
    tc_fence_after();
    {
      float y[64];
      tmem_ld64(t_lane + 0, y);
      float n2 = 0.f;
#pragma unroll
      for (int j = 0; j < 64; ++j) n2 = fmaf(y[j], y[j], n2);
      const float n = sqrtf(n2);
      const float inv = n > 0.f ? 1.0f / n : 0.f;
      unsigned long long cw[3] = {0ull, 0ull, 0ull};  // canonical 192-bit pair-field string: field g at bit 6 g
      float g2 = 0.f;
#pragma unroll
      for (int g = 0; g < 32; ++g) {
        const float u0 = y[2 * g] * inv, u1 = y[2 * g + 1] * inv;
        const int c0 = code_of(u0, thrK), c1 = code_of(u1, thrK);
        const float r0 = u0 - lutK[c0], r1 = u1 - lutK[c1];
        g2 = fmaf(r0, r0, fmaf(r1, r1, g2));
        y[2 * g] = r0 * 8.f, y[2 * g + 1] = r1 * 8.f;  // residual, scaled for the fp16 split (only sign(S r) is used)
        const unsigned long long f = (unsigned long long)(c0 | (c1 << 3));
        const int bit = 6 * g, wi = bit >> 6, sh = bit & 63;
        cw[wi] |= f << sh;
        if (sh > 58) cw[wi + 1] |= f >> (64 - sh);
      }
      // the K MMAs are complete (barrier), so the A buffers can take the residual operands of the S product
#pragma unroll
      for (int kj = 0; kj < 8; ++kj) {
        uint4 hi, lo;
        split8(&y[8 * kj], hi, lo);
        *reinterpret_cast<uint4*>(A_hi + core_off(tid, 8 * kj)) = hi;
        *reinterpret_cast<uint4*>(A_lo + core_off(tid, 8 * kj)) = lo;
      }
      // device layout: the token in slot t stores pair group g at field position (g - t) mod 32, i.e. the canonical
      // string rotated right by 6 t bits; the word part of the rotation goes through shared memory
      unsigned* row = crot + tid * 7;
      row[0] = (unsigned)cw[0], row[1] = (unsigned)(cw[0] >> 32), row[2] = (unsigned)cw[1], row[3] = (unsigned)(cw[1] >> 32);
      row[4] = (unsigned)cw[2], row[5] = (unsigned)(cw[2] >> 32);
      const int wa = (6 * slot) >> 5, wb = (6 * slot) & 31;
      unsigned rw[7];
#pragma unroll
      for (int w = 0; w < 7; ++w) rw[w] = row[(wa + w) % 6];
      if (valid) {
        unsigned o[6];
#pragma unroll
        for (int w = 0; w < 6; ++w) o[w] = __funnelshift_r(rw[w], rw[w + 1], wb);
        *reinterpret_cast<uint4*>(tp + Lo::kOffKC + slot * 16) = make_uint4(o[0], o[1], o[2], o[3]);
        *reinterpret_cast<uint2*>(tp + Lo::kOffKC + 16 * kTile + slot * 8) = make_uint2(o[4], o[5]);
        reinterpret_cast<unsigned short*>(tp + Lo::kOffKN)[slot] = f32_to_f16_bits_clamped(n * inv_sk * 0.0625f);
        reinterpret_cast<unsigned short*>(tp + Lo::kOffKR)[slot] = f32_to_f16_bits_clamped(sqrtf(g2));
      }
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
      gemm(64, aK_hi, bS_hi, true), gemm(64, aK_lo, bS_hi, false), gemm(64, aK_hi, bS_lo, false);
      umma_commit(smem_u32(mbar + 2));
    }
    }  // kKey

    // ---- values: norm, codes; the cache stores V codes per coordinate pair across the 32 tokens of a tile
    if constexpr (!kKey) {
    mbar_wait(smem_u32(mbar + 1), parity);
    tc_fence_after();
    {
      float y[64];
      tmem_ld64(t_lane + 0, y);
      float n2 = 0.f;
#pragma unroll
      for (int j = 0; j < 64; ++j) n2 = fmaf(y[j], y[j], n2);
      const float n = sqrtf(n2);
      const float inv = n > 0.f ? 1.0f / n : 0.f;
#pragma unroll
      for (int g4 = 0; g4 < 8; ++g4) {  // four pair fields per 32-bit shared-memory store
        unsigned w = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int g = 4 * g4 + j;
          const int c0 = code_of(y[2 * g] * inv, thrV), c1 = code_of(y[2 * g + 1] * inv, thrV);
          w |= (unsigned)(c0 | (c1 << 3)) << (8 * j);
        }
        reinterpret_cast<unsigned*>(cbV + tid * 32)[g4] = w;
      }
      if (valid) reinterpret_cast<unsigned short*>(tp + Lo::kOffVN)[slot] = f32_to_f16_bits_clamped(n * inv_sv * 0.0625f);
    }
    __syncthreads();
    {  // thread = (tile of the block, lane = pair group): six words of 32 six-bit fields; tokens of the tile that are
       // outside this call keep their bits (read-modify-write under a mask)
      const int tl = tid >> 5, g = tid & 31;
      const int tile_pos = blk * kBlk + tl * kTile;
      unsigned char* tpv = stream + (size_t)(tile_pos / kTile) * Lo::kTileBytes;
      const int j_first = max(0, a.start_pos - tile_pos), j_end = min(kTile, a.start_pos + a.n_tokens - tile_pos);
      if (j_first < j_end) {
#pragma unroll
        for (int w = 0; w < Lo::KCW; ++w) {
          const int sb = 32 * w;
          unsigned long long word = 0, mask = 0;
#pragma unroll
          for (int j = sb / 6; j <= (sb + 31) / 6 && j < kTile; ++j) {
            if (j < j_first || j >= j_end) continue;
            const unsigned long long f = cbV[(tl * kTile + j) * 32 + g];
            const int sh = 6 * j - sb;
            word |= sh >= 0 ? (f << sh) : (f >> (-sh));
            mask |= sh >= 0 ? (63ull << sh) : (63ull >> (-sh));
          }
          unsigned* p = reinterpret_cast<unsigned*>(tpv + Lo::kOffVC + word_offset(Lo::KCW, w, g));
          const unsigned m32 = (unsigned)mask;
          if (m32 == 0xffffffffu) *p = (unsigned)word;
          else if (m32) *p = (*p & ~m32) | ((unsigned)word & m32);
        }
      }
    }

    }  // !kKey

    // ---- residual sketch: bit j = [(S r)_j >= 0]; nibble group n sits at nibble position (n - t) mod 16
    if constexpr (kKey) {
    mbar_wait(smem_u32(mbar + 2), parity);
    tc_fence_after();
    {
      float y[64];
      tmem_ld64(t_lane + 64, y);
      unsigned long long bits = 0ull;
#pragma unroll
      for (int j = 0; j < 64; ++j) bits |= (unsigned long long)(y[j] >= 0.f ? 1u : 0u) << j;
      const int rs = (4 * slot) & 63;
      const unsigned long long rot = rs ? ((bits >> rs) | (bits << (64 - rs))) : bits;
      if (valid) *reinterpret_cast<uint2*>(tp + Lo::kOffKS + slot * 8) = make_uint2((unsigned)rot, (unsigned)(rot >> 32));
    }
    }  // kKey
    tc_fence_before();  // the next block's MMAs overwrite the accumulators every thread has just read
  }
  __syncthreads();
  if (warp == 0) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(kTmemCols) : "memory");
  }
}

template <typename T>
__global__ void __launch_bounds__(kBlk) quantize_pack_tc_kernel(QuantArgs a, int blocks_per_cta) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  if (blockIdx.z == 0) quantize_pack_tc_body<T, true>(a, blocks_per_cta, smem_dyn);
  else quantize_pack_tc_body<T, false>(a, blocks_per_cta, smem_dyn);
}

template <typename T>
cudaError_t launch_quant_tc_t(const QuantArgs& a, int num_sms, cudaStream_t st) {
  const size_t smem = kSmemBytes;
  const int first_blk = a.start_pos / kBlk, last_blk = (a.start_pos + a.n_tokens - 1) / kBlk;
  const int nblk = last_blk - first_blk + 1;
  const int BH = a.cv.B * a.cv.H;
  const long want = 6L * num_sms;  // per operand (keys / values)  // CTAs: enough to balance the SMs, few enough to amortise staging the matrices
  int bpc = (int)(((long)nblk * BH + want - 1) / want);
  bpc = bpc < 1 ? 1 : (bpc > 16 ? 16 : bpc);
  dim3 grid((nblk + bpc - 1) / bpc, BH, 2);  // z: keys | values
  cudaError_t e = cudaFuncSetAttribute(quantize_pack_tc_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  quantize_pack_tc_kernel<T><<<grid, kBlk, smem, st>>>(a, bpc);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_quantize_pack_tc(const QuantArgs& a, tq_dtype dt, int num_sms, cudaStream_t st) {
  return dt == TQ_F16 ? launch_quant_tc_t<__half>(a, num_sms, st) : launch_quant_tc_t<float>(a, num_sms, st);
}

}  // namespace tq
