// tq_quantize_tc.cu — KV quantize-and-pack on the 5th-generation tensor cores (tcgen05 + TMEM), head_dim 64 and 128.
//
// Same arithmetic as tq_quantize.cu (PAPER.md:111-116 prefill steps 1,3,4; §3.3 Eq. 5; §3.4 Eq. 6 in the sign(S r)
// form of BASELINE.json:north_star), but the three rotations y = PI_K x', S r, PI_V v — a dense
// (tokens x d) x (d x d) contraction — run as tcgen05.mma with the accumulators in tensor memory:
//   * a CTA of 256 (d = 64) / 512 (d = 128) threads owns 128-token blocks of one (batch, head): UMMA M = 128 tokens,
//     N = d outputs, K = 16;
//     keys (RoPE, PI_K, then S on the residual) and values (PI_V) run as separate CTAs (blockIdx.z);
//   * operands are fp16 in shared memory in the canonical K-major no-swizzle layout (8 x 8 core matrices);
//     fp32 accuracy comes from two-term splits a = a_hi + a_lo (each product exact in the fp32 accumulator):
//     D = A_hi B_hi + A_lo B_hi + A_hi B_lo.  Power-of-two scalings keep every split away from the fp16 range
//     limits and cancel exactly: PI x16, the token vector by 2^-exponent(max |x|) (RoPE grows a pair by at most
//     sqrt 2), r x8 (only sign(S r) is used); fp16 values V are exact operands and need two products only.  A numpy
//     study (hard part 4) puts the code-flip rate of this scheme at 2e-7, that of an all-fp32 pipeline;
//   * the prologue is warp-cooperative: a warp stages 8 token rows at a time, lane = (16-byte chunk, row), so that the
//     global reads are sector-exact and the 128-bit shared-memory stores of the operand rows are conflict free;
//   * the epilogue runs d/32 threads per token: thread (token, part) reads the 32 accumulator columns of ITS part of
//     ITS token with ONE tcgen05.ld and keeps them in registers for the norm, the code search, the residual and the
//     packing (the parts exchange their partial sums of squares through shared memory).  The code search and the
//     sign bits are computed on the FMA pipe (see code_f).  The device tile layout (tq_common.cuh) is the A-fragment
//     order of the decode kernel's MMAs, so every thread drops its bytes into an image of the block's four tiles in
//     shared memory (V fields, which mix the two tokens of a pair, are assembled after one shuffle with the neighbour
//     token) and the CTA then writes the image out with coalesced 16-byte stores.  Tiles only partly covered by the
//     call are pre-loaded into the image.
#include "tq_common.cuh"

namespace tq {
namespace {

constexpr int kBlk = 128;      // tokens per block = UMMA M
// d/32 threads per token: thread (token = tid & 127, part = tid >> 7) owns the 32 accumulator columns [32 part, 32 part + 32)
// of its token; 256 threads per CTA at d = 64, 512 at d = 128 (where shared memory allows one CTA per SM: the wider CTA
// doubles the resident warps)
template <int D>
constexpr int kThreadsOf = 128 * (D / 32);

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int D>
struct TcCfg {
  using Lo = Layout<D>;
  static constexpr int kParts = D / 32;            // threads per token
  static constexpr int kThreads = kThreadsOf<D>;
  static constexpr int kSBO = 16 * D;              // bytes between 8-row groups of an operand: 1024 | 2048
  // the A operand of the FIRST product goes through tensor memory as well (stage_rows_tmem): no operand rows in shared
  // memory at all (kTmemA = false keeps the shared-memory path of stage_rows for comparison)
  static constexpr bool kTmemA = true;
  static constexpr int kOpBytes = kTmemA ? 0 : kBlk * D * 2;    // one fp16 A operand in shared memory: 0 | 32 KB
  static constexpr int kMatBytes = D * D * 2;      // one fp16 B operand: 8 | 32 KB
  // tensor memory columns: [0, d) the accumulator (D_K / D_V, then — once every thread holds those in registers — D_S of the
  // residual product); [d, 3d/2) and [3d/2, 2d) the residual operand 8 r as fp16 hi and lo parts (two k per column)
  static constexpr int kTmemCols = 2 * D;
  // instruction descriptor: kind::f16, A = B = fp16 (K-major), D = fp32, N = d, M = 128
  static constexpr uint32_t kIdesc = (1u << 4) | ((uint32_t)(D >> 3) << 17) | ((128u >> 4) << 24);
  // image of one tile's sections owned by a CTA: keys [K codes | K signs | norms k,r], values [V codes | norm v]
  static constexpr int kImgK = Lo::kCodeBytes + Lo::kSignBytes + 4 * kTile;
  static constexpr int kImgV = Lo::kCodeBytes + 2 * kTile;
  static constexpr int kImgBytes = kImgK;          // per tile (the larger of the two)
  // shared memory: B operands 4 x kMatBytes (keys: PI_K hi/lo, S hi/lo; values: PI_V hi/lo) | A operands hi, lo |
  // tile images [4][kImgBytes] | partial sums [2 kinds][d/32 parts][128] | row scales [128] | LUT pair table [64] float2,
  // barriers, TMEM slot
  static constexpr int kOffA = 4 * kMatBytes, kOffMisc = kOffA + 2 * kOpBytes;
  static constexpr int kSmemBytes = kOffMisc + 4 * kImgBytes + 2 * kParts * kBlk * 4 + kBlk * 4 + 64 * 8 + 3 * 8 + 16;
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
// the same with the A operand in tensor memory (lane = row, one 32-bit column per two consecutive k): no shared-memory read
// for A at all
__device__ __forceinline__ void umma_f16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// 16 consecutive 32-bit columns of this thread's TMEM lane, from registers
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
// 16 lanes x 32 columns from the warp's registers in the 16x256b shape: thread t holds, for each of the 4 repeats i, rows
// t / 4 and t / 4 + 8 of the 16 and the columns 8 i + 2 (t % 4), + 1: {row a col 0, row a col 1, row b col 0, row b col 1}
__device__ __forceinline__ void tmem_st_16x256b_x4(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.16x256b.x4.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
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

// NC (32 or 64) consecutive fp32 accumulator columns of this thread's TMEM lane (= its token): every 32-column load is
// issued before the one wait
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
template <int NC>
__device__ __forceinline__ void tmem_ld(uint32_t taddr, float (&v)[NC]) {
  uint32_t r[NC];
#pragma unroll
  for (int c = 0; c < NC / 32; ++c) tmem_ld32_nowait(taddr + 32 * c, r + 32 * c);
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < NC; ++i) v[i] = __uint_as_float(r[i]);
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
  // consecutive threads take consecutive rows n of one 16-byte column chunk: eight of them fill one core matrix row
  // group (128 contiguous bytes), so the 128-bit stores are conflict free; the reads are whole 32-byte sectors
  for (int idx = tid; idx < D * D / 8; idx += kThreadsOf<D>) {
    const int n = idx % D, kj = idx / D;
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

// ---- code search on the FMA pipe ---------------------------------------------------------------------------------------
// code = #{k : u > t_k} for the seven ascending thresholds t_k, u = y / n.  The compare-and-select form (FSETP / FSEL /
// SEL) runs on the half-rate integer ALU pipe, which ncu showed to be the busiest pipe of this kernel (47 %) while the FMA
// pipe idled at 15 %; here the three-step binary search is arithmetic only:
//   [y > T] = sat((y - T) 2^100)  is exactly 0 or 1 (one FFMA.SAT: the fused product-sum has the exact sign, a nonzero
//   difference of two floats of ordinary magnitude times 2^100 exceeds 1, a tie gives 0 = the lower code);
//   the next threshold is picked by multiplying with those 0 / 1 values: T1 + b2 (T5 - T1), and
//   T0 + b1 (T2 - T0) + b2 (T4 - T0) + b1 b2 (T6 - T4 - T2 + T0).
// Everything is compared on the accumulator y against T = t n (n = |y|; 1 for a zero vector, whose codes are those of
// u = 0), so u is never formed.  The picked thresholds are sums of rounded differences and t n is rounded: they differ
// from the fp32 midpoints by a few ulp (relative 2e-7), far inside the 1e-5 band in which a code may differ from the
// fp64 oracle (and of the same size as the rounding of y itself).  Thresholds closer to zero than 2^-70 other than an
// exact 0 would break the 0 / 1 property; Lloyd-Max midpoints are not.
constexpr float kBig = 1.2676506002282294e30f;  // 2^100
struct Search {
  float k3, k1, k51, k0, kA, kB, kC;  // -T 2^100: T3, T1, T5 - T1, T0, T2 - T0, T4 - T0, (T6 - T4) - (T2 - T0)
};
__device__ __forceinline__ Search make_search(const float (&t)[7]) {
  Search s;
  s.k3 = -t[3] * kBig, s.k1 = -t[1] * kBig, s.k51 = -(t[5] - t[1]) * kBig, s.k0 = -t[0] * kBig;
  s.kA = -(t[2] - t[0]) * kBig, s.kB = -(t[4] - t[0]) * kBig;
  s.kC = -((t[6] - t[4]) - (t[2] - t[0])) * kBig;
  return s;
}
__device__ __forceinline__ Search scaled(const Search& c, float nn) {
  return Search{c.k3 * nn, c.k1 * nn, c.k51 * nn, c.k0 * nn, c.kA * nn, c.kB * nn, c.kC * nn};
}
__device__ __forceinline__ float fma_sat(float a, float b, float c) {
  float d;
  asm("fma.rn.sat.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}
// Two coordinates at once: the threshold selection and the code assembly run as packed fp32x2 operations (FFMA2 / FMUL2,
// one instruction for both coordinates; there is no saturating form, so the three comparisons stay scalar): 13
// instructions per pair instead of 20.
struct Search2 {
  float k3;
  float2 k1, k51, k0, kA, kB, kC;  // both halves equal
};
__device__ __forceinline__ Search2 pair_search(const Search& s) {
  return Search2{s.k3, {s.k1, s.k1}, {s.k51, s.k51}, {s.k0, s.k0}, {s.kA, s.kA}, {s.kB, s.kB}, {s.kC, s.kC}};
}
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
  float2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;"
      : "=l"(*reinterpret_cast<unsigned long long*>(&d))
      : "l"(*reinterpret_cast<const unsigned long long*>(&a)), "l"(*reinterpret_cast<const unsigned long long*>(&b)),
        "l"(*reinterpret_cast<const unsigned long long*>(&c)));
  return d;
}
__device__ __forceinline__ float2 fmul2(float2 a, float2 b) {
  float2 d;
  asm("mul.rn.f32x2 %0, %1, %2;"
      : "=l"(*reinterpret_cast<unsigned long long*>(&d))
      : "l"(*reinterpret_cast<const unsigned long long*>(&a)), "l"(*reinterpret_cast<const unsigned long long*>(&b)));
  return d;
}
// the codes of (y0, y1) as floats
__device__ __forceinline__ float2 code_f2(float y0, float y1, const Search2& s) {
  const float2 b2 = make_float2(fma_sat(y0, kBig, s.k3), fma_sat(y1, kBig, s.k3));
  const float2 m1 = ffma2(b2, s.k51, s.k1);
  const float2 b1 = make_float2(fma_sat(y0, kBig, m1.x), fma_sat(y1, kBig, m1.y));
  const float2 m0 = ffma2(fmul2(b1, b2), s.kC, ffma2(b2, s.kB, ffma2(b1, s.kA, s.k0)));
  const float2 b0 = make_float2(fma_sat(y0, kBig, m0.x), fma_sat(y1, kBig, m0.y));
  return ffma2(b2, make_float2(4.f, 4.f), ffma2(b1, make_float2(2.f, 2.f), b0));
}
// an exact small integer held in a float, as an unsigned (F2I runs on the otherwise idle conversion pipe)
__device__ __forceinline__ unsigned f2u(float x) { return __float2uint_rn(x); }


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

// ---- prologue: the A operand rows of one 128-token block -------------------------------------------------------------
// Warp w stages rows [16 w, 16 w + 16) in two groups of 8 (d = 64; [8 w, 8 w + 8) with the 16 warps of d = 128); lane = 8 kk + r owns row r of the group and the 8-value
// chunks kj = kk + 4 i (i < d/32).  A quarter-warp (fixed kk) reads 8 rows x 16 bytes (whole sectors once the other
// chunks of the row are counted) and writes 8 consecutive 16-byte rows of one core matrix: no bank conflict.
// Keys: RoPE from the fp64-evaluated table, power-of-two row scale, two-term split.  Values: fp16 rows are exact
// operands (copied), fp32 rows are scaled and split.  scale_s[row] = the exact inverse row scale.
template <int D, typename T, bool kKey>
__device__ __forceinline__ void stage_rows(const T* __restrict__ src, int i_first /* call index of block row 0 */, int n_tokens,
                                           const float* __restrict__ cs_blk /* rope_cs row of block row 0 */, int rows_cs /* rows of the table left */,
                                           int rope_layout, unsigned char* ahi, unsigned char* alo, float* scale_s, int warp, int lane) {
  constexpr int NI = D / 32;  // chunks per lane and row
  constexpr int GPW = 16 / (kThreadsOf<D> / 32);  // groups of 8 rows per warp: 2 (8 warps) | 1 (16 warps)
  const int r = lane & 7, kk = lane >> 3;
#pragma unroll
  for (int gi = 0; gi < GPW; ++gi) {
    const int row = 8 * GPW * warp + 8 * gi + r;
    const int i = i_first + row;
    const bool valid = i >= 0 && i < n_tokens;
    const T* p = src + (size_t)i * D;
    if constexpr (!kKey && sizeof(T) == 2) {
#pragma unroll
      for (int ii = 0; ii < NI; ++ii) {
        const int kj = kk + 4 * ii;
        *reinterpret_cast<uint4*>(ahi + core_off<D>(row, 8 * kj)) =
            valid ? __ldg(reinterpret_cast<const uint4*>(p) + kj) : make_uint4(0, 0, 0, 0);
      }
      if (kk == 0) scale_s[row] = 1.f;
    } else {
      float x[NI][8];
#pragma unroll
      for (int ii = 0; ii < NI; ++ii) load8<T>(p + 8 * (kk + 4 * ii), valid, x[ii]);
      float amax = 0.f;
#pragma unroll
      for (int ii = 0; ii < NI; ++ii)
#pragma unroll
        for (int j = 0; j < 8; ++j) amax = fmaxf(amax, fabsf(x[ii][j]));
      amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 8));
      amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, 16));
      float s, inv_s;
      pow2_scale(amax, s, inv_s);  // |RoPE(x) s| < 2 sqrt 2
      if (kk == 0) scale_s[row] = inv_s;
      if constexpr (kKey) {
        const float* cs_row = cs_blk + (size_t)min(row, rows_cs - 1) * D;
        if (rope_layout == 0) {  // pairs (2g, 2g+1): four pairs per chunk
#pragma unroll
          for (int ii = 0; ii < NI; ++ii) {
            const int kj = kk + 4 * ii;
            const float4 c0 = __ldg(reinterpret_cast<const float4*>(cs_row + 8 * kj)), c1 = __ldg(reinterpret_cast<const float4*>(cs_row + 8 * kj) + 1);
            const float cs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
            float y[8];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              y[2 * j] = x[ii][2 * j] * cs[2 * j] - x[ii][2 * j + 1] * cs[2 * j + 1];
              y[2 * j + 1] = x[ii][2 * j] * cs[2 * j + 1] + x[ii][2 * j + 1] * cs[2 * j];
            }
            store_split8<D>(y, s, ahi, alo, row, 8 * kj);
          }
        } else {  // pairs (g, g + d/2): chunk kj with chunk kj + d/16, both owned by this lane
#pragma unroll
          for (int ii = 0; ii < NI / 2; ++ii) {
            const int kj = kk + 4 * ii;
            float ya[8], yb[8];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              const float4 c = __ldg(reinterpret_cast<const float4*>(cs_row + 16 * kj) + q);  // pairs g = 8 kj + 2q, + 1
              ya[2 * q] = x[ii][2 * q] * c.x - x[ii + NI / 2][2 * q] * c.y, yb[2 * q] = x[ii][2 * q] * c.y + x[ii + NI / 2][2 * q] * c.x;
              ya[2 * q + 1] = x[ii][2 * q + 1] * c.z - x[ii + NI / 2][2 * q + 1] * c.w;
              yb[2 * q + 1] = x[ii][2 * q + 1] * c.w + x[ii + NI / 2][2 * q + 1] * c.z;
            }
            store_split8<D>(ya, s, ahi, alo, row, 8 * kj);
            store_split8<D>(yb, s, ahi, alo, row, D / 2 + 8 * kj);
          }
        }
      } else {
#pragma unroll
        for (int ii = 0; ii < NI; ++ii) store_split8<D>(x[ii], s, ahi, alo, row, 8 * (kk + 4 * ii));
      }
    }
  }
}

// ---- prologue through tensor memory ------------------------------------------------------------------------------------
// Warp w stages 16 rows x 64 values of the block in the 16x256b shape: rows [32 (w & 3) + 16 (j & 1), + 16) — TMEM lanes it
// may write — and the values k in [64 cj, 64 cj + 64), j = w >> 2, cj = j >> 1 (d = 64: 8 warps, cj = 0; d = 128: 16 warps,
// two warps share a row).  Thread t owns rows t / 4 and t / 4 + 8 of the 16 and, for i = 0..3, the four values
// k = 64 cj + 16 i + 4 (t % 4) .. + 3 (two 32-bit columns of packed fp16 pairs).  A quad reads 32 contiguous bytes of a
// row per load (whole sectors); RoPE pairs (2g, 2g + 1) sit inside a piece; pairs (g, g + d/2) sit in pieces i and i + 2 of
// the same thread at d = 64 and in the other warp of the row at d = 128 (which therefore loads the partner values as
// well); the row maximum is two shuffles, plus one exchange through shared memory at d = 128.  The hi parts go to columns
// [a_col, a_col + d/2), the lo parts to [a_col + d/2, a_col + d).
template <int D, typename T, bool kKey>
__device__ __forceinline__ void stage_rows_tmem(const T* __restrict__ src, int i_first, int n_tokens, const float* __restrict__ cs_blk,
                                                int rows_cs, int rope_layout, uint32_t tmem, uint32_t a_col, float* scale_s,
                                                float* pmax /* [2][128] scratch, d = 128 */, int warp, int lane) {
  const int j = warp >> 2, cj = j >> 1;
  const int row0 = 32 * (warp & 3) + 16 * (j & 1), tq4 = lane & 3, k0 = 64 * cj + 4 * tq4;
  constexpr bool kRaw = !kKey && sizeof(T) == 2;  // fp16 values are exact operands: the raw halves
  uint32_t hi[16], lo[16];
  float x[2][4][4];
  [[maybe_unused]] float xp[2][4][4];  // d = 128, half-split RoPE: the partner values k +- 64
  float amax[2] = {0.f, 0.f};
  const bool split128 = kKey && D == 128 && rope_layout == 1;
  auto load_row = [&](int rb) {  // rows t / 4 (rb = 0) and t / 4 + 8 (rb = 1)
    const int row = row0 + (lane >> 2) + 8 * rb;
    const int i = i_first + row;
    const bool valid = i >= 0 && i < n_tokens;
    const T* p = src + (size_t)i * D + k0;
    if constexpr (kRaw) {
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) {
        const uint2 v = valid ? __ldg(reinterpret_cast<const uint2*>(p + 16 * ii)) : make_uint2(0u, 0u);
        hi[4 * ii + 2 * rb] = v.x, hi[4 * ii + 2 * rb + 1] = v.y;
      }
      if (tq4 == 0 && cj == 0) scale_s[row] = 1.f;
    } else {
      auto load4 = [&](const T* q, float (&o)[4]) {
        if (!valid) {
          o[0] = o[1] = o[2] = o[3] = 0.f;
        } else if constexpr (sizeof(T) == 2) {
          const uint2 v = __ldg(reinterpret_cast<const uint2*>(q));
          const float2 f0 = __half22float2(*reinterpret_cast<const __half2*>(&v.x)), f1 = __half22float2(*reinterpret_cast<const __half2*>(&v.y));
          o[0] = f0.x, o[1] = f0.y, o[2] = f1.x, o[3] = f1.y;
        } else {
          const float4 v = __ldg(reinterpret_cast<const float4*>(q));
          o[0] = v.x, o[1] = v.y, o[2] = v.z, o[3] = v.w;
        }
      };
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) load4(p + 16 * ii, x[rb][ii]);
      if constexpr (D == 128 && kKey) {
        if (split128) {
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) load4(p + 16 * ii + (cj ? -64 : 64), xp[rb][ii]);
        }
      }
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int e = 0; e < 4; ++e) amax[rb] = fmaxf(amax[rb], fabsf(x[rb][ii][e]));
      amax[rb] = fmaxf(amax[rb], __shfl_xor_sync(0xffffffffu, amax[rb], 1));
      amax[rb] = fmaxf(amax[rb], __shfl_xor_sync(0xffffffffu, amax[rb], 2));
      if constexpr (D == 128) {
        if (tq4 == 0) pmax[cj * kBlk + row] = amax[rb];
      }
    }
  };
  auto finish_row = [&](int rb) {
    {
      const int row = row0 + (lane >> 2) + 8 * rb;
      if constexpr (D == 128) amax[rb] = fmaxf(pmax[row], pmax[kBlk + row]);
      float sc, inv_s;
      pow2_scale(amax[rb], sc, inv_s);  // |RoPE(x) s| < 2 sqrt 2
      if (tq4 == 0 && cj == 0) scale_s[row] = inv_s;
      if constexpr (kKey) {
        const float* cs_row = cs_blk + (size_t)min(row, rows_cs - 1) * D;
        if (rope_layout == 0) {  // pairs (2g, 2g + 1): values k, k + 1 use the (cos, sin) at floats [k, k + 2)
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            const float4 c = __ldg(reinterpret_cast<const float4*>(cs_row + k0 + 16 * ii));
            float(&v)[4] = x[rb][ii];
            const float y0 = v[0] * c.x - v[1] * c.y, y1 = v[0] * c.y + v[1] * c.x;
            const float y2 = v[2] * c.z - v[3] * c.w, y3 = v[2] * c.w + v[3] * c.z;
            v[0] = y0, v[1] = y1, v[2] = y2, v[3] = y3;
          }
        } else if constexpr (D == 64) {  // pairs (g, g + 32): pieces ii and ii + 2; pair g uses floats [2 g, 2 g + 2)
#pragma unroll
          for (int ii = 0; ii < 2; ++ii) {
            const float4 c0 = __ldg(reinterpret_cast<const float4*>(cs_row + 2 * (16 * ii + 4 * tq4)));
            const float4 c1 = __ldg(reinterpret_cast<const float4*>(cs_row + 2 * (16 * ii + 4 * tq4)) + 1);
            const float cs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float xa = x[rb][ii][e], xb = x[rb][ii + 2][e];
              x[rb][ii][e] = xa * cs[2 * e] - xb * cs[2 * e + 1];
              x[rb][ii + 2][e] = xa * cs[2 * e + 1] + xb * cs[2 * e];
            }
          }
        } else {  // d = 128, pairs (g, g + 64): this warp holds one member, xp the other; pair g = 16 ii + 4 tq4 + e
#pragma unroll
          for (int ii = 0; ii < 4; ++ii) {
            const float4 c0 = __ldg(reinterpret_cast<const float4*>(cs_row + 2 * (16 * ii + 4 * tq4)));
            const float4 c1 = __ldg(reinterpret_cast<const float4*>(cs_row + 2 * (16 * ii + 4 * tq4)) + 1);
            const float cs[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float xa = cj ? xp[rb][ii][e] : x[rb][ii][e], xb = cj ? x[rb][ii][e] : xp[rb][ii][e];
              x[rb][ii][e] = cj ? xa * cs[2 * e + 1] + xb * cs[2 * e] : xa * cs[2 * e] - xb * cs[2 * e + 1];
            }
          }
        }
      }
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) {
#pragma unroll
        for (int h2 = 0; h2 < 2; ++h2) {
          const float a0 = x[rb][ii][2 * h2] * sc, a1 = x[rb][ii][2 * h2 + 1] * sc;
          const __half2 hh = __floats2half2_rn(a0, a1);
          const float2 hf = __half22float2(hh);
          const __half2 ll = __floats2half2_rn(a0 - hf.x, a1 - hf.y);
          hi[4 * ii + 2 * rb + h2] = *reinterpret_cast<const unsigned*>(&hh);
          lo[4 * ii + 2 * rb + h2] = *reinterpret_cast<const unsigned*>(&ll);
        }
      }
    }
  };
  // d = 64: one row after the other (fewest live registers); d = 128: both rows loaded, the row maxima exchanged between
  // the two warps of a row through shared memory, then both rows finished
  if constexpr (D == 64) {
#pragma unroll
    for (int rb = 0; rb < 2; ++rb) {
      load_row(rb);
      if constexpr (!kRaw) finish_row(rb);
    }
  } else {
    load_row(0), load_row(1);
    if constexpr (!kRaw) {
      __syncthreads();
      finish_row(0), finish_row(1);
    }
  }
  const uint32_t taddr = tmem + ((uint32_t)row0 << 16) + a_col + 32 * cj;
  tmem_st_16x256b_x4(taddr, hi);
  if constexpr (!kRaw) tmem_st_16x256b_x4(taddr + D / 2, lo);
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// kLit: the paper-literal Eq. 6-7 mode (include/tq.h): the accumulator is compared as it stands (no normalisation), the
// norm plane is 1.0 and the rnorm plane the per-head constant e-bar m sqrt(2/pi)
// kVq: the values carry a residual sketch too (tq_shape.v_qjl = 1): the value CTAs then run the S product on 8 r_v and
// drop its sign bits into the V-sketch tile (tq_common.cuh VskLayout), whose image lives in the unused tail of the
// value CTA's tile image
template <int D, typename T, bool kKey, bool kLit, bool kVq>
__device__ __forceinline__ void quantize_pack_tc_body(const QuantArgs& a, int blocks_per_cta, int cta_x, unsigned char* smem) {
  using Cfg = TcCfg<D>;
  using Lo = Layout<D>;
  constexpr bool kF16 = sizeof(T) == 2;
  constexpr int KCW = Lo::KCW, KSW = Lo::KSW;
  constexpr int NC = 32;                       // accumulator columns per thread
  constexpr int kParts = Cfg::kParts, kThreads = Cfg::kThreads;
  unsigned char *B0_hi = smem, *B0_lo = smem + Cfg::kMatBytes;                               // PI_K | PI_V
  unsigned char *B1_hi = smem + 2 * Cfg::kMatBytes, *B1_lo = smem + 3 * Cfg::kMatBytes;      // S (keys only)
  unsigned char *A_hi = smem + Cfg::kOffA, *A_lo = A_hi + Cfg::kOpBytes;
  unsigned char* img = smem + Cfg::kOffMisc;                                  // [4 tiles][kImgBytes]
  float* red_n = reinterpret_cast<float*>(img + 4 * Cfg::kImgBytes);          // [parts][128] partial |y|^2
  float* red_g = red_n + kParts * kBlk;                                       // [parts][128] partial |8 r|^2
  float* scale_s = red_g + kParts * kBlk;                                     // [128] inverse row scales
  float2* lutp = reinterpret_cast<float2*>(scale_s + kBlk);                   // [64] keys: (-8 lut[c0], -8 lut[c1]) at c0 + 8 c1
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(lutp + 64);  // [0]: first product, [1]: S product
  unsigned* tmem_slot = reinterpret_cast<unsigned*>(mbar + 3);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int tok = tid & (kBlk - 1), half = tid >> 7;  // epilogue role: token row and column part ("half" at d = 64)
  auto part_sum = [&](const float* red) {               // the token's sum over the parts, in a fixed order
    float acc = red[tok];
#pragma unroll
    for (int q = 1; q < kParts; ++q) acc += red[q * kBlk + tok];
    return acc;
  };
  const int bh = blockIdx.y, b = bh / a.cv.H, h = bh % a.cv.H;
  const int first_blk = a.start_pos / kBlk, last_blk = (a.start_pos + a.n_tokens - 1) / kBlk;
  const int blk0 = first_blk + cta_x * blocks_per_cta;
  if (blk0 > last_blk) return;
  const int blk1 = min(last_blk, blk0 + blocks_per_cta - 1);
  if (kKey && cta_x == 0 && h == 0 && tid == 0) a.cv.seq_len[a.layer * a.cv.B + b] = a.start_pos + a.n_tokens;

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
    if constexpr (kVq) stage_matrix<D>(B1_hi, B1_lo, a.S, 1.f, tid);
  }
  // thresholds t_k = (lut_k + lut_{k+1}) / 2 in fp32, as search constants; keys also keep a table of LUT pairs for the
  // residual: the S product takes 8 r (only sign(S r) is used, and 8 r splits cleanly in fp16), |r| = |8 r| / 8
  Search search0;
  float lut_cap = 1.f;
  {
    const float* lut_g = (kKey ? a.lut_k : a.lut_v) + h * 8;
    float l8[8], thr[7];
#pragma unroll
    for (int q = 0; q < 8; ++q) l8[q] = __ldg(lut_g + q);
#pragma unroll
    for (int q = 0; q < 7; ++q) thr[q] = 0.5f * (l8[q] + l8[q + 1]);
    search0 = make_search(thr);
    if ((kKey || kVq) && tid < 64) lutp[tid] = make_float2(-8.f * __ldg(lut_g + (tid & 7)), -8.f * __ldg(lut_g + (tid >> 3)));
    if constexpr (kLit) {  // power of two that puts the largest LUT entry in [2^8, 2^9): bound of the residual operand scale
      float s_l, inv_l;
      pow2_scale(fmaxf(fabsf(l8[0]), fabsf(l8[7])), s_l, inv_l);
      lut_cap = s_l * 256.f;
    }
  }
  const unsigned short lit_rnorm = (kLit && kKey) ? literal_rnorm_bits(__ldg(a.ebar_k + h), D) : (unsigned short)0;
  const float lutp_base = (float)smem_u32(lutp);  // shared-window address, exact in fp32
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  // this thread's TMEM lane (its token) and first column: warps w and w + 4 share the lane quadrant w % 4
  const uint32_t t_lane = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(half * NC);
  const uint32_t a_hi = smem_u32(A_hi), a_lo = smem_u32(A_lo), b0_hi = smem_u32(B0_hi), b0_lo = smem_u32(B0_lo),
                 b1_hi = smem_u32(B1_hi), b1_lo = smem_u32(B1_lo);
  auto gemm = [&](uint32_t dcol, uint32_t a_op, uint32_t b_op, bool first) {  // D[:, dcol..dcol+d) (+)= A B^T, K = d
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks)
      umma_f16(tmem + dcol, umma_desc<D>(a_op + ks * 256), umma_desc<D>(b_op + ks * 256), Cfg::kIdesc,
               (first && ks == 0) ? 0u : 1u);
  };

  // the residual product D[:, 0..d) (+)= R S^T with the operand R in tensor memory (column of k-step ks: + 8 ks)
  auto gemm_ts = [&](uint32_t a_col, uint32_t b_op, bool first) {
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks)
      umma_f16_ts(tmem, tmem + a_col + 8 * ks, umma_desc<D>(b_op + ks * 256), Cfg::kIdesc, (first && ks == 0) ? 0u : 1u);
  };
  // this thread's 32 residual values (k = 32 part .. 32 part + 31 of its token) as hi / lo halves into tensor memory
  auto store_residual = [&](const float (&r)[32]) {
    uint32_t hi[16], lo[16];
#pragma unroll
    for (int kj = 0; kj < 4; ++kj) {
      uint4 h4, l4;
      split8(&r[8 * kj], h4, l4);
      hi[4 * kj] = h4.x, hi[4 * kj + 1] = h4.y, hi[4 * kj + 2] = h4.z, hi[4 * kj + 3] = h4.w;
      lo[4 * kj] = l4.x, lo[4 * kj + 1] = l4.y, lo[4 * kj + 2] = l4.z, lo[4 * kj + 3] = l4.w;
    }
    const uint32_t lane_base = tmem + ((uint32_t)((warp & 3) * 32) << 16);
    tmem_st16(lane_base + D + 16 * half, hi);
    tmem_st16(lane_base + D + D / 2 + 16 * half, lo);
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  };
  const T* src = reinterpret_cast<const T*>(kKey ? a.k : a.v) + (size_t)bh * a.n_tokens * D;
  unsigned char* stream = a.cv.tiles + ((size_t)a.layer * a.cv.B * a.cv.H + bh) * a.cv.stream_bytes;
  using Vs = VskLayout<D>;
  unsigned char* vstream = kVq ? a.cv.vsk + ((size_t)a.layer * a.cv.B * a.cv.H + bh) * a.cv.vsk_stream_bytes : nullptr;
  static_assert(Cfg::kImgBytes - Cfg::kImgV >= Vs::kTileBytes, "the V-sketch image fits behind the value image");
  const int slot = tok & 31, tl = tok >> 5, sg = slot & 7, sr = slot >> 3;
  unsigned char* timg = img + tl * Cfg::kImgBytes;  // image of this token's tile
  constexpr int kOffImgKS = Lo::kCodeBytes, kOffImgNK = Lo::kCodeBytes + Lo::kSignBytes;  // keys image
  constexpr int kOffImgVN = Lo::kCodeBytes;                                                // values image
  // byte `sb` of lane l's word string in a section of W words per lane
  // The code section of the IMAGE is not in the order of the tile: inside every [16-byte chunk][lane] array the lane index
  // is permuted so that the byte stores of one warp instruction (32 consecutive tokens, one fixed byte of their fields) land
  // in eight different 16-byte bank groups instead of two (ncu: 4-6 wavefronts per byte store before).  Keys: the eight
  // lanes 4 g + t (g = 0..7) of a fixed t -> g + 8 t; values: lanes 4 gi + tt with (tt, gi >> 2) varying -> tt + 4 (gi >> 2)
  // + 8 (gi & 3).  The copies between image and tile (pre-load, write-out) apply the permutation per 16-byte unit.
  auto perm_lane = [](int l) { return kKey ? (l >> 2) + 8 * (l & 3) : (l & 3) + 4 * (l >> 4) + 8 * ((l >> 2) & 3); };
  // byte `sb` of lane l's word string in the code section (W words per lane) of the image
  auto sec_byte = [&](int W, int l, int sb) {
    const int w = sb >> 2;
    return (w < (W / 4) * 4 ? word_offset(W, w, perm_lane(l)) : word_offset(W, w, l)) + (sb & 3);
  };
  // image offset of the 16-byte unit at byte `ib` of the CTA's share of a tile (code section first, then the rest)
  auto img_unit = [&](int ib) {
    constexpr int kChunked = (KCW / 4) * 16 * kTile;  // bytes of the [chunk][lane] arrays of the code section
    if (ib >= kChunked) return ib;
    const int q = ib >> 4;
    return ((q & ~31) + perm_lane(q & 31)) << 4;
  };

  for (int blk = blk0; blk <= blk1; ++blk) {
    const uint32_t parity = (uint32_t)(blk - blk0) & 1u;
    const int pos = blk * kBlk + tok;
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
      for (int idx = tid; idx < 4 * (kOwn / 16); idx += kThreads) {
        const int t4 = idx / (kOwn / 16), q = idx % (kOwn / 16);
        if (tile_cover(t4) != 1) continue;
        const unsigned char* tg = stream + (size_t)(blk * 4 + t4) * Lo::kTileBytes;
        // keys: [0, kOffVC) then the norms; values: the V codes then |v|
        const int ib = 16 * q;
        const int gb = kKey ? (ib < Lo::kOffVC ? ib : Lo::kOffNK + (ib - Lo::kOffVC))
                            : (ib < Lo::kCodeBytes ? Lo::kOffVC + ib : Lo::kOffVN + (ib - Lo::kCodeBytes));
        *reinterpret_cast<uint4*>(img + t4 * Cfg::kImgBytes + img_unit(ib)) = *reinterpret_cast<const uint4*>(tg + gb);
      }
    }

    if constexpr (!kKey && kVq) {  // V-sketch image: partly covered tiles keep their other tokens' bits, the rest start at zero
      for (int idx = tid; idx < 4 * (Vs::kTileBytes / 16); idx += kThreads) {
        const int t4 = idx / (Vs::kTileBytes / 16), q = idx % (Vs::kTileBytes / 16);
        uint4 v = make_uint4(0, 0, 0, 0);
        if (tile_cover(t4) == 1) v = *reinterpret_cast<const uint4*>(vstream + (size_t)(blk * 4 + t4) * Vs::kTileBytes + 16 * q);
        *reinterpret_cast<uint4*>(img + t4 * Cfg::kImgBytes + Cfg::kImgV + 16 * q) = v;
      }
    }
    // ---- stage the A operand rows of the block and start the first product
    {
      const int p0 = blk * kBlk;  // cache position (= RoPE position) of block row 0
      if constexpr (Cfg::kTmemA)
        stage_rows_tmem<D, T, kKey>(src, p0 - a.start_pos, a.n_tokens, a.rope_cs + (size_t)min(p0, a.cv.max_seq - 1) * D,
                                    a.cv.max_seq - min(p0, a.cv.max_seq - 1), a.rope_layout, tmem, D, scale_s, red_g, warp, lane);
      else
        stage_rows<D, T, kKey>(src, p0 - a.start_pos, a.n_tokens, a.rope_cs + (size_t)min(p0, a.cv.max_seq - 1) * D,
                               a.cv.max_seq - min(p0, a.cv.max_seq - 1), a.rope_layout, A_hi, A_lo, scale_s, warp, lane);
    }
    if constexpr (!Cfg::kTmemA) fence_async_smem();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
      tc_fence_after();
      if constexpr (Cfg::kTmemA) {
        gemm_ts(D, b0_hi, true), gemm_ts(D, b0_lo, false);
        if (kKey || !kF16) gemm_ts(D + D / 2, b0_hi, false);
      } else {
        gemm(0, a_hi, b0_hi, true), gemm(0, a_hi, b0_lo, false);
        if (kKey || !kF16) gemm(0, a_lo, b0_hi, false);
      }
      umma_commit(smem_u32(mbar + 0));
    }
    if (tid == 32 && blk < blk1) {  // the next block's input rows on their way to L2 while this block is worked on
      const int lo = max((blk + 1) * kBlk - a.start_pos, 0), hi = min((blk + 2) * kBlk - a.start_pos, a.n_tokens);
      if (hi > lo)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src + (size_t)lo * D), "r"((unsigned)((hi - lo) * D * sizeof(T))) : "memory");
    }
    mbar_wait(smem_u32(mbar + 0), parity);
    tc_fence_after();

    // ---- thread = (token, column half): its d/2 accumulator columns, once; |y|^2 through shared memory
    float y[NC];
    tmem_ld<NC>(t_lane, y);
    {
      float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f;
#pragma unroll
      for (int j = 0; j < NC; j += 4) {
        p0 = fmaf(y[j], y[j], p0), p1 = fmaf(y[j + 1], y[j + 1], p1);
        p2 = fmaf(y[j + 2], y[j + 2], p2), p3 = fmaf(y[j + 3], y[j + 3], p3);
      }
      red_n[half * kBlk + tok] = (p0 + p1) + (p2 + p3);
    }
    __syncthreads();
    const float n = sqrtf(part_sum(red_n));
    const float row_scale = 16.f / scale_s[tok];  // y = 16 s PI x, s a power of two
    const unsigned short n_h = kLit ? kF16One : f32_to_f16_bits_clamped(n * scale_s[tok] * 0.0625f);
    // thresholds on the accumulator scale: t |y| for the unit vector, t 16 s for the activation itself (literal mode)
    const Search sr_n = scaled(search0, kLit ? row_scale : (n > 0.f ? n : 1.f));
    const Search2 sr_2 = pair_search(sr_n);

    if constexpr (kKey) {
      // ---- codes, residual (the A operand of the S product, written over this token's operand row: the first product is
      //      complete).  Pair p = half d/4 + g belongs to lane (sg, t = g & 3) as field j = half d/32 + (g >> 2) of this
      //      token's block, bits [6 (J sr + j), + 6) of the lane's string: four fields = three bytes
      const float inv8 = n > 0.f ? 8.0f / n : 0.f;
      // literal mode: residual operand = rs (y_true - lut[c]) with the power of two rs = min(16 s, lut_cap), so that
      // neither term leaves the fp16 range whatever the scale of the row
      const float rs = fminf(row_scale, lut_cap), rA = rs / row_scale, rB = rs * 0.125f;
      float2 g2 = make_float2(0.f, 0.f);
      const float2 inv8_2 = make_float2(inv8, inv8);
      float yt[4][NC / 32];  // four six-bit fields = one 24-bit word, accumulated exactly in fp32
#pragma unroll
      for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int wi = 0; wi < NC / 32; ++wi) yt[t][wi] = 0.f;
#pragma unroll
      for (int g = 0; g < NC / 2; ++g) {
        const float2 cc = code_f2(y[2 * g], y[2 * g + 1], sr_2);
        const float field = fmaf(cc.y, 8.f, cc.x);  // c0 | c1 << 3
        float2 nl;  // (-8 lut[c0], -8 lut[c1])
        asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(nl.x), "=f"(nl.y) : "r"(f2u(fmaf(field, 8.f, lutp_base))));
        float2 rr;
        if constexpr (kLit) rr = ffma2(make_float2(y[2 * g], y[2 * g + 1]), make_float2(rA, rA), fmul2(nl, make_float2(rB, rB)));
        else rr = ffma2(make_float2(y[2 * g], y[2 * g + 1]), inv8_2, nl);  // 8 (u - lut[c])
        g2 = ffma2(rr, rr, g2);
        y[2 * g] = rr.x, y[2 * g + 1] = rr.y;
        yt[g & 3][g >> 4] = fmaf(field, (float)(1u << (6 * ((g >> 2) & 3))), yt[g & 3][g >> 4]);
      }
      red_g[half * kBlk + tok] = g2.x + g2.y;
      if (valid) {
#pragma unroll
        for (int t = 0; t < 4; ++t)
#pragma unroll
          for (int wi = 0; wi < NC / 32; ++wi) {
            const int sb = (6 * Lo::J * sr) / 8 + 3 * (half * (NC / 32) + wi);  // byte of the lane's K string
            const unsigned w24 = f2u(yt[t][wi]);
#pragma unroll
            for (int k = 0; k < 3; ++k) timg[sec_byte(KCW, 4 * sg + t, sb + k)] = (unsigned char)(w24 >> (8 * k));
          }
      }
      store_residual(y);
      tc_fence_before();
      __syncthreads();
      if (tid == 0) {
        tc_fence_after();
        gemm_ts(D, b1_hi, true), gemm_ts(D + D / 2, b1_hi, false), gemm_ts(D, b1_lo, false);
        umma_commit(smem_u32(mbar + 1));
      }
      if (valid && half == 0)
        reinterpret_cast<unsigned*>(timg + kOffImgNK)[slot_lane(slot)] =
            (unsigned)n_h |
            ((unsigned)(kLit ? lit_rnorm : f32_to_f16_bits_clamped(sqrtf(part_sum(red_g)) * 0.125f)) << 16);
      // ---- residual sketch: bit j = [(S r)_j >= 0] for this thread's sketch rows [half d/2, + d/2).  Sketch rows
      //      [t d/4, (t+1) d/4) belong to lane (sg, t) as 16-bit pieces u; a piece is stored as two bytes of word (mt, u):
      //      byte (sr & 1) holds bits 0..7, byte 2 + (sr & 1) bits 8..15 (the byte interleave with the slot 8 further on
      //      makes the decode kernel's fp16x2 masks work)
      mbar_wait(smem_u32(mbar + 1), parity);
      tc_fence_after();
      tmem_ld<NC>(t_lane, y);  // D_S took the accumulator columns
#pragma unroll
      for (int c = 0; c < NC / 32; ++c) {
        // [y >= 0] = sat(y 2^100 + 1), sixteen bits summed exactly in one float
        float2 w01 = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const float pw = (float)(1u << j);
          w01 = ffma2(make_float2(fma_sat(y[32 * c + j], kBig, 1.f), fma_sat(y[32 * c + 16 + j], kBig, 1.f)), make_float2(pw, pw), w01);
        }
        const unsigned w = f2u(w01.x) | (f2u(w01.y) << 16);
        if (valid) {
#pragma unroll
          for (int q = 0; q < 2; ++q) {
            const int rho0 = half * NC + 32 * c + 16 * q, t = rho0 / (D / 4), u = (rho0 % (D / 4)) >> 4;
            const int word = (sr >> 1) * Lo::U + u;
            unsigned char* wp = timg + kOffImgKS + word_offset(KSW, word, 4 * sg + t);
            wp[sr & 1] = (unsigned char)(w >> (16 * q));
            wp[2 + (sr & 1)] = (unsigned char)(w >> (16 * q + 8));
          }
        }
      }
    } else {
      // ---- values: codes of this thread's coordinates, eight per word; one shuffle hands them to the neighbour token
      //      of the pair, then the pair assembles the six-bit fields code_i(even token) | code_i(odd token) << 3 of lane
      //      (i & 7, pp & 3), block j = pp >> 2: the even token builds the lanes i & 7 < 4, the odd one the others.
      //      This thread's coordinates 8 c + (i & 7), c in [half d/16, + d/16), are d/16 fields = 3 d/64 bytes per lane
      constexpr int CW = NC / 8;  // coordinates 8 c + q, c < CW, of this thread
      // F[q] = sum_c code(8 c + q) 64^c: the token's three-bit halves of the CW six-bit fields of lane q, exact in fp32
      float F[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) F[q] = 0.f;
      [[maybe_unused]] const float inv8 = n > 0.f ? 8.0f / n : 0.f;
      [[maybe_unused]] float g2a = 0.f, g2b = 0.f;
#pragma unroll
      for (int c = 0; c < CW; ++c) {
        if constexpr (kVq) {  // pairs of coordinates share one look-up of (-8 lut[c0], -8 lut[c1]); y becomes 8 r_v
#pragma unroll
          for (int q = 0; q < 8; q += 2) {
            const float2 cc = code_f2(y[8 * c + q], y[8 * c + q + 1], sr_2);
            const float c0 = cc.x, c1 = cc.y;
            F[q] = fmaf(c0, (float)(1u << (6 * c)), F[q]), F[q + 1] = fmaf(c1, (float)(1u << (6 * c)), F[q + 1]);
            float2 nl;
            asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(nl.x), "=f"(nl.y) : "r"(f2u(fmaf(fmaf(c1, 8.f, c0), 8.f, lutp_base))));
            const float r0 = fmaf(y[8 * c + q], inv8, nl.x), r1 = fmaf(y[8 * c + q + 1], inv8, nl.y);
            g2a = fmaf(r0, r0, g2a), g2b = fmaf(r1, r1, g2b);
            y[8 * c + q] = r0, y[8 * c + q + 1] = r1;
          }
        } else {
#pragma unroll
          for (int q = 0; q < 8; q += 2) {
            const float2 cc = code_f2(y[8 * c + q], y[8 * c + q + 1], sr_2);
            F[q] = fmaf(cc.x, (float)(1u << (6 * c)), F[q]), F[q + 1] = fmaf(cc.y, (float)(1u << (6 * c)), F[q + 1]);
          }
        }
      }
      if constexpr (kVq) {  // the residual operand of the S product over this token's operand row
        red_g[half * kBlk + tok] = g2a + g2b;
        store_residual(y);
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {
          tc_fence_after();
          gemm_ts(D, b1_hi, true), gemm_ts(D + D / 2, b1_hi, false), gemm_ts(D, b1_lo, false);
          umma_commit(smem_u32(mbar + 1));
        }
      }
      if (valid && half == 0) reinterpret_cast<unsigned short*>(timg + kOffImgVN)[slot_lane(slot)] = n_h;
      {
        // the even token of a pair builds the lanes gi = 0..3, the odd one 4..7: each hands the other the four F it needs,
        // field word = F(even token) + 8 F(odd token), 24 bits = three bytes of lane (gi, pp & 3)'s string
        const int e = slot & 1, pp = slot >> 1;
        const bool v_partner = __shfl_xor_sync(0xffffffffu, (int)valid, 1) != 0;
        const bool v_e = e ? v_partner : valid, v_o = e ? valid : v_partner;
        float recv[4];
#pragma unroll
        for (int gq = 0; gq < 4; ++gq) recv[gq] = __shfl_xor_sync(0xffffffffu, e ? F[gq] : F[4 + gq], 1);
        if (v_e || v_o) {
          constexpr int NB = 6 * CW / 8;  // bytes per (lane, token pair, column part): 3
          // bits of the even token inside three consecutive bytes of a field string (period 24 bits)
          constexpr unsigned kEvenMask[3] = {0xC7u, 0x71u, 0x1Cu};
#pragma unroll
          for (int gq = 0; gq < 4; ++gq) {
            const int gi = 4 * e + gq;
            const float own = e ? F[4 + gq] : F[gq];
            const unsigned acc = f2u(e ? fmaf(own, 8.f, recv[gq]) : fmaf(recv[gq], 8.f, own));
            const int sb0 = (pp >> 2) * (6 * Lo::C / 8) + half * NB;  // byte of the lane's V string
#pragma unroll
            for (int k = 0; k < NB; ++k) {
              unsigned char* dst = timg + sec_byte(KCW, 4 * gi + (pp & 3), sb0 + k);
              const unsigned char nb = (unsigned char)(acc >> (8 * k));
              if (v_e && v_o) {
                *dst = nb;
              } else {  // partial pair: keep the other token's bits
                const unsigned char m = (unsigned char)(v_e ? kEvenMask[k % 3] : ~kEvenMask[k % 3]);
                *dst = (unsigned char)((*dst & ~m) | (nb & m));
              }
            }
          }
        }
      }
    }
    if constexpr (!kKey && kVq) {
      // ---- V-side sketch: bit [(S r_v)_rho >= 0] of this thread's sketch rows [half d/2, + d/2) goes to lane
      //      (rho & 7, t of the slot), one word per (thread, lane): the token's old bits are cleared, the new ones set
      unsigned char* vimg = timg + Cfg::kImgV;
      if (valid && half == 0)
        reinterpret_cast<unsigned short*>(vimg + Vs::kOffVR)[slot_lane(slot)] =
            f32_to_f16_bits_clamped(sqrtf(part_sum(red_g)) * 0.125f);
      mbar_wait(smem_u32(mbar + 1), parity);
      tc_fence_after();
      tmem_ld<NC>(t_lane, y);  // D_S took the accumulator columns
      if (valid) {
        const int ks = slot >> 4, th = (slot >> 3) & 1, ts = (slot & 7) >> 1, e = slot & 1;
        const int word = ks * (D / 64) + (half >> 1);  // the two m-tiles of this thread's rows (2 part, 2 part + 1) share one word
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          unsigned bits = 0u, own = 0u;
#pragma unroll
          for (int mq = 0; mq < NC / 16; ++mq)  // m-tile half NC/16 + mq, row halves rh
#pragma unroll
            for (int rh = 0; rh < 2; ++rh) {
              const int mt = half * (NC / 16) + mq;
              const unsigned pos = 16u * e + 4u * (mt & 3) + 2u * rh + th;
              own |= 1u << pos;
              bits |= (y[16 * mq + 8 * rh + g] >= 0.f ? 1u : 0u) << pos;
            }
          unsigned* wp = reinterpret_cast<unsigned*>(vimg + Vs::kOffVS + word_offset(Vs::KSW, word, 4 * g + ts));
          atomicAnd(wp, ~own);
          atomicOr(wp, bits);
        }
      }
    }
    // ---- write the block's tile images out (every tile the call touches; the image of a partly covered tile carries
    //      the old bits of the other tokens)
    __syncthreads();
    if constexpr (!kKey && kVq) {
      for (int idx = tid; idx < 4 * (Vs::kTileBytes / 16); idx += kThreads) {
        const int t4 = idx / (Vs::kTileBytes / 16), q = idx % (Vs::kTileBytes / 16);
        if (tile_cover(t4) == 0) continue;
        *reinterpret_cast<uint4*>(vstream + (size_t)(blk * 4 + t4) * Vs::kTileBytes + 16 * q) =
            *reinterpret_cast<const uint4*>(img + t4 * Cfg::kImgBytes + Cfg::kImgV + 16 * q);
      }
    }
    {
      constexpr int kOwn = kKey ? Cfg::kImgK : Cfg::kImgV;
      for (int idx = tid; idx < 4 * (kOwn / 16); idx += kThreads) {
        const int t4 = idx / (kOwn / 16), q = idx % (kOwn / 16);
        if (tile_cover(t4) == 0) continue;
        unsigned char* tg = stream + (size_t)(blk * 4 + t4) * Lo::kTileBytes;
        const int ib = 16 * q;
        const int gb = kKey ? (ib < Lo::kOffVC ? ib : Lo::kOffNK + (ib - Lo::kOffVC))
                            : (ib < Lo::kCodeBytes ? Lo::kOffVC + ib : Lo::kOffVN + (ib - Lo::kCodeBytes));
        *reinterpret_cast<uint4*>(tg + gb) = *reinterpret_cast<const uint4*>(img + t4 * Cfg::kImgBytes + img_unit(ib));
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

// grid = (block groups, batch x heads, keys | values): the key CTAs (the long ones) are dispatched first and the value
// CTAs fill in behind them (measured: alternating key and value CTAs along x is 8 % slower at configs[2])
constexpr int kQuantCtasPerSm64 = 4;  // 64 registers: four CTAs per SM also fill tensor memory (4 x 128 columns); measured 147 us vs 158 us with three
template <int D, typename T, bool kLit, bool kVq>
__global__ void __launch_bounds__(kThreadsOf<D>, D == 64 ? kQuantCtasPerSm64 : 1) quantize_pack_tc_kernel(QuantArgs a, int blocks_per_cta) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  if (blockIdx.z == 0) quantize_pack_tc_body<D, T, true, kLit, kVq>(a, blocks_per_cta, (int)blockIdx.x, smem_dyn);
  else quantize_pack_tc_body<D, T, false, kLit, kVq>(a, blocks_per_cta, (int)blockIdx.x, smem_dyn);
}

template <int D, typename T, bool kLit, bool kVq>
cudaError_t launch_quant_tc_t(const QuantArgs& a, int num_sms, cudaStream_t st) {
  const size_t smem = TcCfg<D>::kSmemBytes;
  const int first_blk = a.start_pos / kBlk, last_blk = (a.start_pos + a.n_tokens - 1) / kBlk;
  const int nblk = last_blk - first_blk + 1;
  const int BH = a.cv.B * a.cv.H;
  const long want = 4L * num_sms;  // CTAs per operand: enough to balance the SMs, few enough to amortise the matrices
  int bpc = (int)(((long)nblk * BH + want - 1) / want);
  bpc = bpc < 1 ? 1 : (bpc > 16 ? 16 : bpc);
  dim3 grid((nblk + bpc - 1) / bpc, BH, 2);  // z: keys | values
  cudaError_t e = cudaFuncSetAttribute(quantize_pack_tc_kernel<D, T, kLit, kVq>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  quantize_pack_tc_kernel<D, T, kLit, kVq><<<grid, kThreadsOf<D>, smem, st>>>(a, bpc);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

template <bool kLit, bool kVq>
static cudaError_t launch_quant_tc_mode(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st) {
  if (D == 64)
    return dt == TQ_F16 ? launch_quant_tc_t<64, __half, kLit, kVq>(a, num_sms, st) : launch_quant_tc_t<64, float, kLit, kVq>(a, num_sms, st);
  return dt == TQ_F16 ? launch_quant_tc_t<128, __half, kLit, kVq>(a, num_sms, st) : launch_quant_tc_t<128, float, kLit, kVq>(a, num_sms, st);
}

cudaError_t launch_quantize_pack_tc(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st) {
  if (a.literal) return launch_quant_tc_mode<true, false>(a, D, dt, num_sms, st);
  if (a.cv.vsk) return launch_quant_tc_mode<false, true>(a, D, dt, num_sms, st);
  return launch_quant_tc_mode<false, false>(a, D, dt, num_sms, st);
}

}  // namespace tq
