// tq_decode.cu — fused decode attention over the packed 3-bit cache (sm_100a).
//
// Algorithm 1 of the paper re-associated as BASELINE.json:north_star asks: the query is
// rotated once (q'' = PI_K RoPE(q), z = S q''; Eq. 4 moves PI from every key to the query), then the cache
// is streamed exactly once:
//   logit_j = n_j ( <q'', lut_K[codes_j]> + sqrt(pi/2)/m * g_j * <z, sigma_j> ) / sqrt(d)
//   online softmax (running max m, sum l), o' += p_j * nv_j * lut_V[codesV_j];   out = PI_V^T (o' / l).
//
// Why warp-level tensor-core MMAs (DESIGN.md §5.1 has the counters): the round-1 kernel did these three
// contractions with per-unit shared-memory tables of partial dot products and CUDA-core adds; ncu showed it bound by
// the shared-memory pipe (LSU 49 %) and the integer ALU (46 %) at 36 % of the HBM roofline — 70 % of the roofline
// would have needed more than 95 % of both.  Here a lookup only DEQUANTISES (a 64-entry table of fp16 pairs
// (lut[c0], lut[c1]) that does not depend on the query), and the multiply-accumulate runs on mma.sync.m16n8k16
// (fp16 x fp16 -> fp32), which is otherwise idle:
//   * K scores : A = dequantised key codes (16 tokens x 16 coordinates per MMA), B = q'' split hi + lo in fp16 in
//                the columns of B (both products exact in the fp32 accumulator);
//   * sign term: A = the stored sign bits themselves: (word & (0x00010001 << p)) is an fp16x2 register whose halves
//                are 0 or the subnormal 2^(p-24) (mma.sync multiplies fp16 subnormals exactly); B = z scaled by
//                2^(E-p), so the accumulator holds 2^(E-24) sum_j bit_j z_j and <z, sigma> = 2 sum - sum(z);
//   * V        : A = dequantised value codes (16 coordinates x 16 tokens), B = the softmax weights split hi + lo.
// The tile layout (tq_common.cuh) stores every word in A-fragment order, so a lookup is SHF + LOP3 + LDS and needs no
// cross-lane traffic; the table column is the lane, so no lookup ever has a bank conflict.
// The fp16 tables are exact when the LUT entries are binary16-representable (tq_calibrate_host emits such LUTs:
// DESIGN.md reading D15); any other fp32 LUT takes the two-term path (hi + lo tables, twice the MMAs).
//
// Staging: every warp owns a ring of kStages tile slots in shared memory filled by cp.async.bulk (1-D TMA copy,
// mbarrier complete_tx); lane 0 re-arms a slot as soon as the warp has consumed it.
// Split-K over the sequence: grid = units x nsplit CTAs; a unit covered by one CTA is finished in place, otherwise the
// last CTA to arrive merges the partial (m, l, o') triples.  Either way the finishing CTA applies PI_V^T.
#include <utility>

#include "tq_common.cuh"

namespace tq {

constexpr int kMaxSegments = 64;      // split-K partial slots per unit (tq_api.cu sizes the workspace)
constexpr int kDecodeCtasPerSm64 = 5;  // d = 64 without the V sketch: 96 registers, 36 KB shared memory
constexpr int kDecodeThreads = 128;   // warps of one CTA share the dequantisation tables of one head
constexpr int kDecodeWarps = kDecodeThreads / 32;
constexpr int kStages = 2;  // tile slots per warp (measured at configs[2] x 33 layers: 2 slots 11.4 us per layer, 3 slots 11.5, 4 slots 13.2)

// Shared-memory map in ABSOLUTE shared-window addresses: the table and ring bases are immediates of the ld.shared
// instructions, so a lookup address is one LOP3 ((field & mask) | lane * 4).  Dynamic shared memory starts right after
// the 1 KB the driver reserves; the kernel traps if the window starts later than kAbsMisc.
// kVq: the values carry a residual sketch (tq_shape.v_qjl = 1): every ring slot also holds the tile of the V-sketch stream
// and the per-warp / per-split records carry the sketch accumulator b[m] and the weight sum W'
template <int D, bool kVq = false>
struct DecodeCfg {
  using Lo = Layout<D>;
  using Vs = VskLayout<D>;
  static constexpr int kSlotBytes = Lo::kTileBytes + (kVq ? Vs::kTileBytes : 0);
  static constexpr int kRec = kVq ? 2 * D + 3 : D + 2;  // floats of one (m, l, o'[D] [, b[D], W']) record
  static constexpr unsigned kAbsMisc = 1024;   // mbarriers [warps][kStages], weights [warps][2][32] halves, flag
  static constexpr unsigned kAbsBar = kAbsMisc;
  static constexpr unsigned kAbsWbuf = kAbsMisc + 128;  // per warp [hi | lo][32] halves of w, then the same of w'
  static constexpr unsigned kAbsFlag = kAbsWbuf + kDecodeWarps * 256;
  static constexpr unsigned kAbsRed = 2304;    // per-warp records then the merged o [2 D] and t [D]
  static constexpr int kRedBytes = kDecodeWarps * kRec * 4 + 3 * D * 4;
  static constexpr unsigned kAbsRing = (kAbsRed + kRedBytes + 127) / 128 * 128;
  static constexpr int kRingBytes = kDecodeWarps * kStages * kSlotBytes;
  static constexpr unsigned kAbsTab = (kAbsRing + kRingBytes + 255) / 256 * 256;  // K table then V table
  // bytes per table: [64 entries][32 lanes] fp16 pairs, or [64][16] (hi pair, lo pair) for LUTs that are not
  // binary16-representable (64-bit reads are served one half-warp at a time, so 16 columns are conflict free)
  static constexpr int kTabBytes = 64 * 32 * 4;
  static constexpr int kSmemBytes = kAbsTab + 2 * kTabBytes;  // requested dynamic bytes (window start <= 1 KB)
  static constexpr int kCtasPerSm = D == 64 ? (kVq ? 4 : kDecodeCtasPerSm64) : 2;
};

// ---- small PTX helpers --------------------------------------------------------------------------------------------
template <unsigned BASE>
__device__ __forceinline__ unsigned lds_u32(unsigned addr) {
  unsigned v;  // not volatile: the tables are constant once built, the scheduler may hoist and interleave lookups
  asm("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(addr), "n"(BASE));
  return v;
}
template <unsigned BASE>
__device__ __forceinline__ uint2 lds_u32x2(unsigned addr) {
  uint2 v;
  asm("ld.shared.v2.u32 {%0, %1}, [%2+%3];" : "=r"(v.x), "=r"(v.y) : "r"(addr), "n"(BASE));
  return v;
}
__device__ __forceinline__ uint4 lds_u32x4(unsigned addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ uint2 lds_u32x2_dyn(unsigned addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void mma16816(float (&d)[4], unsigned a0, unsigned a1, unsigned a2, unsigned a3, unsigned b0,
                                         unsigned b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mbar_init(unsigned bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred P1;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// one 1-D TMA copy of `bytes` (multiple of 16) global -> shared, completion counted on the mbarrier
__device__ __forceinline__ void tma_load_tile(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}

// the same for a main tile and its V-sketch tile: two copies into one slot, one transaction count
__device__ __forceinline__ void tma_load_tile2(unsigned dst, const void* src, unsigned bytes, const void* src2, unsigned bytes2,
                                               unsigned bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes + bytes2) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst + bytes),
               "l"(src2), "r"(bytes2), "r"(bar)
               : "memory");
}

// bits [BIT, BIT+NB) of the little-endian word string w, moved to bit position LS and masked
template <int LS, int BIT, int NB, int NW>
__device__ __forceinline__ unsigned field_at(const unsigned (&w)[NW]) {
  constexpr int wi = BIT >> 5, s = BIT & 31;
  constexpr unsigned mask = ((1u << NB) - 1u) << LS;
  unsigned v;
  if constexpr (s + NB > 32)
    v = __funnelshift_r(w[wi], w[(wi + 1) % NW], (s - LS) & 31);
  else if constexpr (s >= LS)
    v = w[wi] >> (s - LS);
  else
    v = w[wi] << (LS - s);
  return v & mask;
}

__device__ __forceinline__ float ex2_ftz(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float warp_max_f32(float x) {  // sm_100a: one CREDUX instead of five shuffles
  float y;
  asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ unsigned pack_h2(__half lo, __half hi) {
  return (unsigned)__half_as_ushort(lo) | ((unsigned)__half_as_ushort(hi) << 16);
}
// x = hi + lo in binary16 (two-term split; exact to 2^-22 |x| while |x| stays in the normal range)
__device__ __forceinline__ void split_h(float x, __half& hi, __half& lo) {
  hi = __float2half_rn(x);
  lo = __float2half_rn(x - __half2float(hi));
}
__device__ __forceinline__ bool f16_exact(float x) { return __half2float(__float2half_rn(x)) == x; }
// 2^e as a float, e in [-126, 127]
__device__ __forceinline__ float pow2i(int e) { return __uint_as_float((unsigned)(e + 127) << 23); }
// exponent e with 2^e <= |x| < 2^(e+1) (0 for zero / denormal / non-finite input)
__device__ __forceinline__ int exponent_of(float x) {
  const int E = (int)((__float_as_uint(x) >> 23) & 0xffu);
  return (E == 0 || E == 255) ? 0 : E - 127;
}

// ---- the per-unit B operands ------------------------------------------------------------------------------------------
// The prep kernel leaves q'' log2(e)/sqrt(d) and z log2(e)/sqrt(d) sqrt(pi/2)/m as fp32 in the workspace.  Every lane
// builds the B fragments it feeds to the MMAs: column n of B holds the hi part for even n and the lo part for odd n, so a
// lane's accumulator pair (columns 2t, 2t+1) sums to the full product for every t: no cross-lane traffic afterwards.
template <int D>
struct UnitFrags {
  unsigned bq[D / 16][2];  // K scores: k-step ks, registers b0 (coordinates 16 ks + 2t, +1), b1 (+8, +9)
  unsigned bz[D / 16][2];  // sign term
  float kscale;            // accumulator -> <q'', lut> in log2 units
  float sscale, zsum;      // accumulator -> 2 sum_j bit_j z_j ; sum_j z_j
};

// this lane's pattern (g & 1, t) of the unit's fragment block (tq_common.cuh FragLayout), four 128-bit loads per 16 words
template <int D>
__device__ __forceinline__ void load_frags(UnitFrags<D>& f, const unsigned* fb, int lane) {
  using FL = FragLayout<D>;
  constexpr int KS = D / 16;
  const uint4* src = reinterpret_cast<const uint4*>(fb + (((lane >> 2) & 1) * 4 + (lane & 3)) * FL::kWordsPerPat);
  unsigned w[4 * KS];
#pragma unroll
  for (int i = 0; i < KS; ++i) {
    const uint4 v = __ldcg(src + i);
    w[4 * i] = v.x, w[4 * i + 1] = v.y, w[4 * i + 2] = v.z, w[4 * i + 3] = v.w;
  }
  const float4 sc = __ldcg(reinterpret_cast<const float4*>(fb + FL::kScalOff));
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    f.bq[ks][0] = w[2 * ks], f.bq[ks][1] = w[2 * ks + 1];
    f.bz[ks][0] = w[2 * KS + 2 * ks], f.bz[ks][1] = w[2 * KS + 2 * ks + 1];
  }
  f.kscale = sc.x, f.sscale = sc.y, f.zsum = sc.z;
}

// ---- one 32-token tile ------------------------------------------------------------------------------------------------
// kFast: the LUT entries are binary16-representable, the tables hold fp16 pairs (one 32-bit read per field);
// otherwise they hold (hi pair, lo pair) and every field costs one 64-bit read and two MMAs.
template <int D, bool kFast, bool kVq>
struct TileMath {
  using Lo = Layout<D>;
  using Cfg = DecodeCfg<D, kVq>;
  static constexpr int KS = D / 16;       // k-steps of the K / sign contractions
  static constexpr int MV = D / 16;       // m-tiles (16 coordinates each) of the V contraction
  static constexpr int LS = 7;            // log2 of the table row pitch (32 lanes x 4 bytes | 16 x 8 bytes)
  static constexpr unsigned kAbsKtab = Cfg::kAbsTab;
  static constexpr unsigned kAbsVtab = Cfg::kAbsTab + Cfg::kTabBytes;

  // scores of this lane's four token slots: kacc[mt] / sacc[mt] = {row g: hi, lo; row g+8: hi, lo} of m-tile mt
  template <int... KSI>
  static __device__ __forceinline__ void scores(const unsigned (&kw)[Lo::KCW], const unsigned (&sw)[Lo::KSW],
                                                const UnitFrags<D>& f, unsigned lane_off, float (&kacc)[2][4],
                                                float (&sacc)[2][4], std::integer_sequence<int, KSI...>) {
    (([&] {
       constexpr int ks = KSI;
#pragma unroll
       for (int mt = 0; mt < 2; ++mt) {
         // K: fields (r = 2 mt | 2 mt + 1, j = 2 ks | 2 ks + 1) at bit 6 (J r + j)
         const unsigned x0 = fieldk<2 * 0 + 0, ks>(kw, mt) | lane_off, x1 = fieldk<1, ks>(kw, mt) | lane_off;
         const unsigned x2 = fieldk<2, ks>(kw, mt) | lane_off, x3 = fieldk<3, ks>(kw, mt) | lane_off;
         if constexpr (kFast) {
           mma16816(kacc[mt], lds_u32<kAbsKtab>(x0), lds_u32<kAbsKtab>(x1), lds_u32<kAbsKtab>(x2), lds_u32<kAbsKtab>(x3),
                    f.bq[ks][0], f.bq[ks][1]);
         } else {
           const uint2 a0 = lds_u32x2<kAbsKtab>(x0), a1 = lds_u32x2<kAbsKtab>(x1), a2 = lds_u32x2<kAbsKtab>(x2),
                       a3 = lds_u32x2<kAbsKtab>(x3);
           mma16816(kacc[mt], a0.x, a1.x, a2.x, a3.x, f.bq[ks][0], f.bq[ks][1]);
           mma16816(kacc[mt], a0.y, a1.y, a2.y, a3.y, f.bq[ks][0], f.bq[ks][1]);
         }
         // signs: word (mt, u), rows {p0, p0 + 8} and {p0 + 1, p0 + 9} of piece u as fp16 subnormals
         constexpr int u = ks >> 2, p0 = 2 * (ks & 3);
         const unsigned w = sw[mt * Lo::U + u], wb = w >> 8;
         mma16816(sacc[mt], w & (0x00010001u << p0), wb & (0x00010001u << p0), w & (0x00010001u << (p0 + 1)),
                  wb & (0x00010001u << (p0 + 1)), f.bz[ks][0], f.bz[ks][1]);
       }
     }()),
     ...);
  }
  // A register index q (0..3) of (mt, ks): r = 2 mt + (q & 1), j = 2 ks + (q >> 1)
  template <int Q, int KSI>
  static __device__ __forceinline__ unsigned fieldk(const unsigned (&kw)[Lo::KCW], int mt) {
    constexpr int j = 2 * KSI + (Q >> 1);
    return mt == 0 ? field_at<LS, 6 * (Lo::J * (Q & 1) + j), 6>(kw) : field_at<LS, 6 * (Lo::J * (2 + (Q & 1)) + j), 6>(kw);
  }

  // V accumulate for the 16 tokens of k-step KSV: o[mt] += A(16 coordinates x 16 tokens) w
  template <int KSV, int... MTI>
  static __device__ __forceinline__ void values(const unsigned (&vw)[Lo::KCW], unsigned lane_off, unsigned b0, unsigned b1,
                                                float (&o)[MV][4], std::integer_sequence<int, MTI...>) {
    (([&] {
       constexpr int mt = MTI;
       // fields (j = 2 ksv | 2 ksv + 1, c = 2 mt | 2 mt + 1) at bit 6 (C j + c)
       const unsigned x0 = field_at<LS, 6 * (Lo::C * (2 * KSV) + 2 * mt), 6>(vw) | lane_off;
       const unsigned x1 = field_at<LS, 6 * (Lo::C * (2 * KSV) + 2 * mt + 1), 6>(vw) | lane_off;
       const unsigned x2 = field_at<LS, 6 * (Lo::C * (2 * KSV + 1) + 2 * mt), 6>(vw) | lane_off;
       const unsigned x3 = field_at<LS, 6 * (Lo::C * (2 * KSV + 1) + 2 * mt + 1), 6>(vw) | lane_off;
       if constexpr (kFast) {
         mma16816(o[mt], lds_u32<kAbsVtab>(x0), lds_u32<kAbsVtab>(x1), lds_u32<kAbsVtab>(x2), lds_u32<kAbsVtab>(x3), b0, b1);
       } else {
         const uint2 a0 = lds_u32x2<kAbsVtab>(x0), a1 = lds_u32x2<kAbsVtab>(x1), a2 = lds_u32x2<kAbsVtab>(x2),
                     a3 = lds_u32x2<kAbsVtab>(x3);
         mma16816(o[mt], a0.x, a1.x, a2.x, a3.x, b0, b1);
         mma16816(o[mt], a0.y, a1.y, a2.y, a3.y, b0, b1);
       }
     }()),
     ...);
  }
};

// words of a section of W words per lane, from the tile image in shared memory
template <int W>
__device__ __forceinline__ void lds_words(unsigned (&dst)[W], unsigned sec, int lane) {
#pragma unroll
  for (int c = 0; c < W / 4; ++c) {
    const uint4 v = lds_u32x4(sec + c * 16 * kTile + lane * 16);
    dst[4 * c] = v.x, dst[4 * c + 1] = v.y, dst[4 * c + 2] = v.z, dst[4 * c + 3] = v.w;
  }
  if constexpr (W % 4 == 2) {
    const uint2 v = lds_u32x2_dyn(sec + (W / 4) * 16 * kTile + lane * 8);
    dst[W - 2] = v.x, dst[W - 1] = v.y;
  }
}

// ---- the streaming loop of one warp -----------------------------------------------------------------------------------
template <int D, bool kFast, bool kVq>
__device__ __forceinline__ void stream_tiles(const unsigned char* stream, const unsigned char* vstream, int tile_first, int tile1, int T,
                                             int warp, int lane, const UnitFrags<D>& f, float& m_out, float& l_out,
                                             float (&o)[D / 16][4], float (&ob)[D / 16][4], float& wsum_out) {
  using Lo = Layout<D>;
  using Vs = VskLayout<D>;
  using Cfg = DecodeCfg<D, kVq>;
  using TM = TileMath<D, kFast, kVq>;
  constexpr int NW = kDecodeWarps;
  const int t = lane & 3;
  const unsigned lane_off = kFast ? (unsigned)lane << 2 : (unsigned)(lane & 15) << 3;  // table column of this lane
  const unsigned ring = Cfg::kAbsRing + warp * kStages * Cfg::kSlotBytes;
  const unsigned bar0 = Cfg::kAbsBar + warp * kStages * 8;
  const unsigned wbuf = Cfg::kAbsWbuf + warp * 256;  // [hi | lo][32 slots] binary16 of w, then of w'
  const int my_slot = lane_slot(lane);
  float m = -INFINITY, l = 0.f, wsum = 0.f;

  // ring state: slot image and barrier of the tile at hand, phase parity of this round over the ring, and the global
  // address of the tile kStages rounds ahead
  unsigned img = ring, bar = bar0, parity = 0;
  int st = 0;
  const unsigned char* src_next = stream + (size_t)(tile_first + kStages * NW) * Lo::kTileBytes;
  [[maybe_unused]] const unsigned char* vsrc_next = kVq ? vstream + (size_t)(tile_first + kStages * NW) * Vs::kTileBytes : nullptr;
  for (int tile = tile_first; tile < tile1; tile += NW) {
    mbar_wait(bar, parity);

    // ---- scores (tensor cores): lane (g, t) ends up with the K and sign sums of slots g + 8 r
    unsigned kw[Lo::KCW], sw[Lo::KSW];
    lds_words<Lo::KCW>(kw, img + Lo::kOffKC, lane);
    lds_words<Lo::KSW>(sw, img + Lo::kOffKS, lane);
    float kacc[2][4], sacc[2][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) kacc[i][j] = 0.f, sacc[i][j] = 0.f;
    TM::scores(kw, sw, f, lane_off, kacc, sacc, std::make_integer_sequence<int, D / 16>{});
    // this lane's own slot g + 8 t: m-tile t >> 1, row half t & 1
    const float k01 = t & 2 ? kacc[1][0] + kacc[1][1] : kacc[0][0] + kacc[0][1];
    const float k23 = t & 2 ? kacc[1][2] + kacc[1][3] : kacc[0][2] + kacc[0][3];
    const float s01 = t & 2 ? sacc[1][0] + sacc[1][1] : sacc[0][0] + sacc[0][1];
    const float s23 = t & 2 ? sacc[1][2] + sacc[1][3] : sacc[0][2] + sacc[0][3];
    const float kval = (t & 1 ? k23 : k01) * f.kscale;
    const float sval = fmaf(t & 1 ? s23 : s01, f.sscale, -f.zsum);

    // ---- online softmax, lane = token slot
    unsigned nk;
    unsigned short nv;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(nk) : "r"(img + Lo::kOffNK + lane * 4) : "memory");
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(nv) : "r"(img + Lo::kOffVN + lane * 2) : "memory");
    const bool valid = tile * kTile + my_slot < T;
    float s2 = f16_bits_to_f32((unsigned short)(nk & 0xffffu)) * fmaf(f16_bits_to_f32((unsigned short)(nk >> 16)), sval, kval);
    s2 = valid ? s2 : -INFINITY;
    const float mnew = fmaxf(m, warp_max_f32(s2));  // finite: slot 0 of every processed tile is valid
    const float fsc = ex2_ftz(m - mnew);            // 0 on a warp's first tile (m = -inf)
    const float p = ex2_ftz(s2 - mnew);             // invalid lanes: exp2(-inf) = 0
    l = fmaf(l, fsc, p);
    if (mnew != m) {  // warp-uniform
#pragma unroll
      for (int i = 0; i < D / 16; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) o[i][j] *= fsc;
      if constexpr (kVq) {
#pragma unroll
        for (int i = 0; i < D / 16; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) ob[i][j] *= fsc;
      }
    }
    m = mnew;
    const float wv = valid ? p * f16_bits_to_f32(nv) : 0.f;
    [[maybe_unused]] float wq = 0.f;  // w' = w |r_v|: the weight of this token's value sign bits
    if constexpr (kVq) {
      unsigned short gv;
      asm volatile("ld.shared.u16 %0, [%1];" : "=h"(gv) : "r"(img + Lo::kTileBytes + Vs::kOffVR + lane * 2) : "memory");
      wq = valid ? wv * f16_bits_to_f32(gv) : 0.f;  // slots past seq_len may hold any bits (0 x NaN would poison the unit)
      wsum = fmaf(wsum, fsc, wq);
    }
    const unsigned nz = __ballot_sync(0xffffffffu, wv != 0.f);
    if (nz) {
      // hand the weights from lane = slot to the B-fragment order (tokens 2t, 2t+1, 2t+8, 2t+9 of each k-step) through
      // shared memory, split hi + lo: lanes with even g feed the hi column, odd g the lo column
      __half wh, wl;
      split_h(wv, wh, wl);
      __syncwarp();
      asm volatile("st.shared.u16 [%0], %1;" ::"r"(wbuf + my_slot * 2), "h"(__half_as_ushort(wh)) : "memory");
      asm volatile("st.shared.u16 [%0], %1;" ::"r"(wbuf + 64 + my_slot * 2), "h"(__half_as_ushort(wl)) : "memory");
      if constexpr (kVq) {  // tokens of the upper half of a k-step sit one bit higher in the sign words: halve their weight
        __half qh, ql;
        split_h((my_slot & 8) ? 0.5f * wq : wq, qh, ql);
        asm volatile("st.shared.u16 [%0], %1;" ::"r"(wbuf + 128 + my_slot * 2), "h"(__half_as_ushort(qh)) : "memory");
        asm volatile("st.shared.u16 [%0], %1;" ::"r"(wbuf + 192 + my_slot * 2), "h"(__half_as_ushort(ql)) : "memory");
      }
      __syncwarp();
      unsigned vw[Lo::KCW];
      lds_words<Lo::KCW>(vw, img + Lo::kOffVC, lane);
      const unsigned wsrc = wbuf + ((lane >> 2) & 1) * 64 + t * 4;
      // slots 16 ks .. 16 ks + 15 belong to the lanes with (t >> 1) == ks
      if (nz & 0x33333333u) {
        unsigned b0, b1;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(b0) : "r"(wsrc) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+16];" : "=r"(b1) : "r"(wsrc) : "memory");
        TM::template values<0>(vw, lane_off, b0, b1, o, std::make_integer_sequence<int, D / 16>{});
      }
      if (nz & 0xccccccccu) {
        unsigned b0, b1;
        asm volatile("ld.shared.u32 %0, [%1+32];" : "=r"(b0) : "r"(wsrc) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+48];" : "=r"(b1) : "r"(wsrc) : "memory");
        TM::template values<1>(vw, lane_off, b0, b1, o, std::make_integer_sequence<int, D / 16>{});
      }
      if constexpr (kVq) {
        // ---- value sign bits: ob[mt] += bits (16 sketch rows x 16 tokens of k-step ks) x w'; word ks (D/64) + (mt >> 2),
        //      bit 4 (mt & 3) + {0: row g, 2: row g + 8} + {0: tokens 2t, 2t+1; 1: tokens 2t+8, 2t+9} (+16 for the odd token)
        unsigned vsw[Vs::KSW];
        lds_words<Vs::KSW>(vsw, img + Lo::kTileBytes + Vs::kOffVS, lane);
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) {
          if (!(nz & (ks == 0 ? 0x33333333u : 0xccccccccu))) continue;
          unsigned b0, b1;
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(b0) : "r"(wsrc + 128 + 32 * ks) : "memory");
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(b1) : "r"(wsrc + 128 + 32 * ks + 16) : "memory");
#pragma unroll
          for (int mt = 0; mt < D / 16; ++mt) {
            // the upper byte of each half is brought down first: only bits 0..9 of an fp16 are plain 2^(p - 24) subnormals
            const unsigned wd = (mt & 2) ? vsw[ks * (D / 64) + (mt >> 2)] >> 8 : vsw[ks * (D / 64) + (mt >> 2)];
            const int p0 = 4 * (mt & 1);
            mma16816(ob[mt], wd & (0x00010001u << p0), wd & (0x00010001u << (p0 + 2)), wd & (0x00010001u << (p0 + 1)),
                     wd & (0x00010001u << (p0 + 3)), b0, b1);
          }
        }
      }
    }
    // ---- the slot is consumed (every word of the image has been used): refill it with the tile kStages rounds ahead
    __syncwarp();
    if (lane == 0 && tile + kStages * NW < tile1) {
      if constexpr (kVq) tma_load_tile2(img, src_next, Lo::kTileBytes, vsrc_next, Vs::kTileBytes, bar);
      else tma_load_tile(img, src_next, Lo::kTileBytes, bar);
    }
    src_next += NW * Lo::kTileBytes;
    if constexpr (kVq) vsrc_next += NW * Vs::kTileBytes;
    img += Cfg::kSlotBytes, bar += 8;
    if (++st == kStages) st = 0, img = ring, bar = bar0, parity ^= 1u;
  }
  m_out = m;
  l_out = l;
  wsum_out = wsum;
}

// ---- the streaming kernel ------------------------------------------------------------------------------------
// grid = units x nsplit.  CTA (unit uc, split sp) streams tiles [sp * per, (sp + 1) * per) of its unit, per = tiles per
// split planned on the host from t_hint (the last split also takes whatever lies beyond); a shorter cache simply
// leaves the trailing splits empty.  The four warps take tiles round-robin.
// kFusedOut: the finishing CTA applies PI_V^T and writes `out` (per-layer calls); otherwise it leaves o'/l in the
// workspace and finish_kernel rotates every unit of the step at once (tq_decode_model_step).
template <int D, typename TIO, bool kFusedOut, bool kVq>
__global__ void __launch_bounds__(kDecodeThreads, DecodeCfg<D, kVq>::kCtasPerSm) decode_main_kernel(DecodeArgs a) {
  using Lo = Layout<D>;
  using Vs = VskLayout<D>;
  using Cfg = DecodeCfg<D, kVq>;
  constexpr int NW = kDecodeWarps, REC = Cfg::kRec;
  extern __shared__ unsigned char smem_raw[];
  const unsigned raw = (unsigned)__cvta_generic_to_shared(smem_raw);
  if (raw > Cfg::kAbsMisc) __trap();  // the fixed shared-memory map does not fit: fail loudly
  unsigned char* abs0 = smem_raw - raw;  // generic pointer to absolute shared address 0 of this CTA's window
  float* red = reinterpret_cast<float*>(abs0 + Cfg::kAbsRed);  // NW records
  float* omerged = red + NW * REC;                              // [D] + [D] partial matvec
  [[maybe_unused]] float* tmerged = omerged + 2 * D;            // [D] sketch vector t = 2 b - W'
  int* flag = reinterpret_cast<int*>(abs0 + Cfg::kAbsFlag);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // grid = (nsplit, H, layers_in_call x B): no integer division on the way to the unit
  const int B = a.cv.B, H = a.cv.H;
  const int nsplit = (int)gridDim.x, sp = (int)blockIdx.x, h = (int)blockIdx.y, e = (int)blockIdx.z;
  const int lc = a.n_layers_call == 1 ? 0 : e / B, b = e - lc * B;  // e = (layer-in-call, batch); seq_len is contiguous over e
  const int uc = e * H + h;
  const int layer = a.layer_begin + lc;
  const size_t lh = (size_t)layer * H + h;
  const int per = a.per, tile0 = sp * per;
  const int cap1 = sp == nsplit - 1 ? a.cv.tiles_cap : min(a.cv.tiles_cap, tile0 + per);  // static bound of this split
  const unsigned char* stream = a.cv.tiles + (((size_t)layer * B + b) * H + h) * a.cv.stream_bytes;
  [[maybe_unused]] const unsigned char* vstream = kVq ? a.cv.vsk + (((size_t)layer * B + b) * H + h) * a.cv.vsk_stream_bytes : nullptr;

  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < kStages; ++i) mbar_init(Cfg::kAbsBar + (warp * kStages + i) * 8, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const float* Pv = a.pi_v + lh * D * D;
  if constexpr (kFusedOut) {  // a hint: PI_V towards L2 for the epilogue
#pragma unroll
    for (int i = 0; i < D * D * 4 / 128 / kDecodeThreads; ++i)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(Pv + (size_t)(i * kDecodeThreads + tid) * 32));
  }

  if (a.chain_mode == 0) pdl_wait();
  pdl_trigger();  // the launch behind this one may be scheduled: it either waits for this grid or belongs to the same chain
  // ---- the first kStages tiles of this warp go on their way at once (their addresses follow from the host's split
  //      plan alone); the cache length and the unit's B operands are fetched while they fly
  int issued = 0;
#pragma unroll
  for (int i = 0; i < kStages; ++i) issued += (tile0 + warp + i * NW < cap1) ? 1 : 0;
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < kStages; ++i) {
      const int tl = tile0 + warp + i * NW;
      if (tl < cap1) {
        if constexpr (kVq)
          tma_load_tile2(Cfg::kAbsRing + (warp * kStages + i) * Cfg::kSlotBytes, stream + (size_t)tl * Lo::kTileBytes, Lo::kTileBytes,
                         vstream + (size_t)tl * Vs::kTileBytes, Vs::kTileBytes, Cfg::kAbsBar + (warp * kStages + i) * 8);
        else
          tma_load_tile(Cfg::kAbsRing + (warp * kStages + i) * Lo::kTileBytes, stream + (size_t)tl * Lo::kTileBytes, Lo::kTileBytes,
                        Cfg::kAbsBar + (warp * kStages + i) * 8);
      }
    }
  }
  int T;
  asm volatile("ld.global.cg.b32 %0, [%1];" : "=r"(T) : "l"(a.cv.seq_len + a.layer_begin * B + e) : "memory");
  // dequantisation tables of this head (prep kernel): warp w expands entries 16 w .. 16 w + 15 over the lane columns
  const unsigned* tb = a.tabs + ((size_t)lc * H + h) * kTabWords;
  const bool fast = __ldcg(tb + 256) != 0u;
  {
    unsigned kt[16], vt[16];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const uint4 k4 = __ldcg(reinterpret_cast<const uint4*>(tb + warp * 16) + i);
      const uint4 v4 = __ldcg(reinterpret_cast<const uint4*>(tb + 128 + warp * 16) + i);
      kt[4 * i] = k4.x, kt[4 * i + 1] = k4.y, kt[4 * i + 2] = k4.z, kt[4 * i + 3] = k4.w;
      vt[4 * i] = v4.x, vt[4 * i + 1] = v4.y, vt[4 * i + 2] = v4.z, vt[4 * i + 3] = v4.w;
    }
    if (fast) {  // [64][32 lanes] fp16 pairs
      unsigned* kd = reinterpret_cast<unsigned*>(abs0 + Cfg::kAbsTab) + warp * 16 * 32 + lane;
      unsigned* vd = reinterpret_cast<unsigned*>(abs0 + Cfg::kAbsTab + Cfg::kTabBytes) + warp * 16 * 32 + lane;
#pragma unroll
      for (int i = 0; i < 16; ++i) kd[i * 32] = kt[i], vd[i * 32] = vt[i];
    } else {  // [64][16] (hi pair, lo pair)
      uint2* kd = reinterpret_cast<uint2*>(abs0 + Cfg::kAbsTab) + warp * 16 * 16 + (lane & 15);
      uint2* vd = reinterpret_cast<uint2*>(abs0 + Cfg::kAbsTab + Cfg::kTabBytes) + warp * 16 * 16 + (lane & 15);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const uint4 k4 = __ldcg(reinterpret_cast<const uint4*>(tb + 64 + warp * 16) + i);
        const uint4 v4 = __ldcg(reinterpret_cast<const uint4*>(tb + 192 + warp * 16) + i);
        kd[(4 * i) * 16] = make_uint2(kt[4 * i], k4.x), kd[(4 * i + 1) * 16] = make_uint2(kt[4 * i + 1], k4.y);
        kd[(4 * i + 2) * 16] = make_uint2(kt[4 * i + 2], k4.z), kd[(4 * i + 3) * 16] = make_uint2(kt[4 * i + 3], k4.w);
        vd[(4 * i) * 16] = make_uint2(vt[4 * i], v4.x), vd[(4 * i + 1) * 16] = make_uint2(vt[4 * i + 1], v4.y);
        vd[(4 * i + 2) * 16] = make_uint2(vt[4 * i + 2], v4.z), vd[(4 * i + 3) * 16] = make_uint2(vt[4 * i + 3], v4.w);
      }
    }
  }
  UnitFrags<D> fr;
  load_frags<D>(fr, a.frags + (size_t)uc * FragLayout<D>::kWords, lane);
  const int nt = (T + kTile - 1) / kTile;
  const int tile1 = min(nt, cap1);
  const int nseg = min(nsplit, (nt + per - 1) / per);  // splits of this unit that have work
  // every copy that was started must land before this CTA may leave (its shared memory is recycled): the streaming loop
  // consumes the tiles below tile1, the rest is drained here
  {
    const int mine = tile0 + warp < tile1 ? (tile1 - tile0 - warp + NW - 1) / NW : 0;  // tiles this warp will stream
    for (int i = mine; i < issued; ++i) mbar_wait(Cfg::kAbsBar + (warp * kStages + i) * 8, 0u);
  }
  if (tile0 >= nt) {  // empty cache (the prep kernel wrote out = 0) or a trailing split with nothing to do
    if (a.chain_mode != 0) pdl_wait();
    return;
  }
  __syncthreads();  // tables

  float o[D / 16][4];
#pragma unroll
  for (int i = 0; i < D / 16; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) o[i][j] = 0.f;
  float ob[D / 16][4];  // sketch accumulator (kVq)
#pragma unroll
  for (int i = 0; i < D / 16; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) ob[i][j] = 0.f;
  float m, l, wsum;
  if (fast) stream_tiles<D, true, kVq>(stream, vstream, tile0 + warp, tile1, T, warp, lane, fr, m, l, o, ob, wsum);
  else stream_tiles<D, false, kVq>(stream, vstream, tile0 + warp, tile1, T, warp, lane, fr, m, l, o, ob, wsum);

  // ---- reduce over the CTA's warps.  o[mt] = {coordinate 16 mt + g: hi, lo; coordinate 16 mt + g + 8: hi, lo}, the same
  //      in all four lanes of a quad
  l = warp_sum(l);
  if constexpr (kVq) wsum = warp_sum(wsum);
  float* wr = red + warp * REC;
  if (lane == 0) {
    wr[0] = m;
    wr[1] = l;
    if constexpr (kVq) wr[2 + 2 * D] = wsum;
  }
  if ((lane & 3) == 0) {
    const int g = lane >> 2;
#pragma unroll
    for (int mt = 0; mt < D / 16; ++mt) {
      wr[2 + 16 * mt + g] = o[mt][0] + o[mt][1];
      wr[2 + 16 * mt + g + 8] = o[mt][2] + o[mt][3];
      if constexpr (kVq) {  // undo the 2^(p - 24) of the sign bits: row g sat at bit 4 (mt & 1), row g + 8 two bits higher
        wr[2 + D + 16 * mt + g] = (ob[mt][0] + ob[mt][1]) * pow2i(24 - 4 * (mt & 1));
        wr[2 + D + 16 * mt + g + 8] = (ob[mt][2] + ob[mt][3]) * pow2i(22 - 4 * (mt & 1));
      }
    }
  }
  __syncthreads();
  float M = -INFINITY;
#pragma unroll
  for (int w = 0; w < NW; ++w) M = fmaxf(M, red[w * REC]);
  float Lsum = 0.f, oi = 0.f, bi = 0.f, Wq = 0.f;  // bi: sketch accumulator row tid; Wq: sum of the sketch weights
  if (tid < D) {
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const float mw = red[w * REC];
      const float fw = mw == -INFINITY ? 0.f : ex2_ftz(mw - M);
      Lsum = fmaf(red[w * REC + 1], fw, Lsum);
      oi = fmaf(red[w * REC + 2 + tid], fw, oi);
      if constexpr (kVq) {
        bi = fmaf(red[w * REC + 2 + D + tid], fw, bi);
        Wq = fmaf(red[w * REC + 2 + 2 * D], fw, Wq);
      }
    }
  }
  if (nseg > 1) {
    float* part = a.partials + ((size_t)uc * kMaxSegments + sp) * REC;
    if (tid < D) {
      part[2 + tid] = oi;
      if constexpr (kVq) part[2 + D + tid] = bi;
    }
    if (tid == 0) {
      part[0] = M;
      part[1] = Lsum;
      if constexpr (kVq) part[2 + 2 * D] = Wq;
    }
    __syncthreads();
    if (tid == 0) {  // release: the barrier orders the CTA's partial stores before this fence (cumulativity)
      __threadfence();
      const int old = atomicAdd(&a.counters[uc], 1);
      *flag = (old == nseg - 1);
      if (old == nseg - 1) a.counters[uc] = 0;
      __threadfence();  // acquire side for the CTA that merges
    }
    __syncthreads();
    if (*flag == 0) {
      if (a.chain_mode != 0) pdl_wait();
      return;
    }
    const float* pp = a.partials + (size_t)uc * kMaxSegments * REC;
    M = -INFINITY;
    for (int s = 0; s < nseg; ++s) M = fmaxf(M, __ldcg(pp + s * REC));
    Lsum = 0.f;
    oi = 0.f, bi = 0.f, Wq = 0.f;
    if (tid < D) {
      for (int s = 0; s < nseg; ++s) {
        const float ms = __ldcg(pp + s * REC);
        const float fs = ms == -INFINITY ? 0.f : ex2_ftz(ms - M);
        Lsum = fmaf(__ldcg(pp + s * REC + 1), fs, Lsum);
        oi = fmaf(__ldcg(pp + s * REC + 2 + tid), fs, oi);
        if constexpr (kVq) {
          bi = fmaf(__ldcg(pp + s * REC + 2 + D + tid), fs, bi);
          Wq = fmaf(__ldcg(pp + s * REC + 2 + 2 * D), fs, Wq);
        }
      }
    }
  }
  if constexpr (kVq) {
    // ---- o' += sqrt(pi/2)/m S^T t, t = sum_j w'_j sigma_j = 2 b - W' (sigma = 2 bits - 1): thread i owns coordinate i and
    //      column i of S (coalesced over the CTA)
    if (tid < D) tmerged[tid] = 2.f * bi - Wq;
    __syncthreads();
    if (tid < D) {
      float acc0 = 0.f, acc1 = 0.f;
#pragma unroll 8
      for (int rho = 0; rho < D; rho += 2) {
        acc0 = fmaf(__ldg(a.S + (size_t)rho * D + tid), tmerged[rho], acc0);
        acc1 = fmaf(__ldg(a.S + (size_t)(rho + 1) * D + tid), tmerged[rho + 1], acc1);
      }
      oi = fmaf(acc0 + acc1, (D == 64 ? 0.01958303339555469f : 0.009791516697777345f), oi);  // sqrt(pi/2) / m
    }
  }
  if constexpr (!kFusedOut) {
    if (tid < D) a.orot[(size_t)uc * D + tid] = Lsum > 0.f ? oi / Lsum : 0.f;
  } else {
    // ---- out = PI_V^T (o' / l): the k range is split over the 128 / D thread groups; every load is issued before the
    //      first multiply (one L2 round trip), four independent chains per thread
    if (tid < D) omerged[tid] = Lsum > 0.f ? oi / Lsum : 0.f;
    __syncthreads();
    constexpr int PARTS = kDecodeThreads / D;  // 2 | 1
    constexpr int KP = D / PARTS;              // 32 | 128
    const int i = tid % D, part = (tid / D) % PARTS;
    float r = 0.f;
    {
      const float* Pvp = Pv + (size_t)part * KP * D + i;
#pragma unroll
      for (int k0 = 0; k0 < KP; k0 += 32) {
        float pv[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) pv[k] = __ldg(Pvp + (size_t)(k0 + k) * D);
        float r0 = 0.f, r1 = 0.f, r2 = 0.f, r3 = 0.f;
#pragma unroll
        for (int k = 0; k < 32; k += 4) {
          r0 = fmaf(pv[k], omerged[part * KP + k0 + k], r0);
          r1 = fmaf(pv[k + 1], omerged[part * KP + k0 + k + 1], r1);
          r2 = fmaf(pv[k + 2], omerged[part * KP + k0 + k + 2], r2);
          r3 = fmaf(pv[k + 3], omerged[part * KP + k0 + k + 3], r3);
        }
        r += (r0 + r1) + (r2 + r3);
      }
    }
    if (PARTS > 1 && part > 0) omerged[part * D + i] = r;
    __syncthreads();
    if (tid < D) {
#pragma unroll
      for (int pp = 1; pp < PARTS; ++pp) r += omerged[pp * D + i];
      TIO* outp = reinterpret_cast<TIO*>(a.out) + (size_t)uc * D;
      if constexpr (sizeof(TIO) == 2) outp[i] = __float2half_rn(r);
      else outp[i] = r;
    }
  }
  if (a.chain_mode != 0) pdl_wait();  // complete in launch order (see DecodeArgs::chain_mode)
}

// ---- out = PI_V^T orot for every unit of a model step (tq_decode_model_step): one CTA per (layer-in-call, head) and
//      group of kFinB batch entries; thread i owns output coordinate i and column i of PI_V (coalesced over the CTA)
constexpr int kFinB = 8;
template <int D, typename TIO>
__global__ void __launch_bounds__(D) finish_kernel(DecodeArgs a, int nbg) {
  __shared__ float os[kFinB][D];
  const int i = threadIdx.x, B = a.cv.B, H = a.cv.H;
  const int bgi = (int)blockIdx.x % nbg, lh_c = (int)blockIdx.x / nbg, lc = lh_c / H, h = lh_c - lc * H;
  const int b0 = bgi * kFinB, nb = min(kFinB, B - b0);
  const float* Pv = a.pi_v + ((size_t)(a.layer_begin + lc) * H + h) * D * D;
  // launched with programmatic stream serialization: PI_V is a constant of the call, so its first 32 rows are fetched
  // while the last streaming kernels of the chain are still running; only orot has to wait for them
  float pv[32];
#pragma unroll
  for (int k = 0; k < 32; ++k) pv[k] = __ldg(Pv + (size_t)k * D + i);
  pdl_wait();
#pragma unroll
  for (int e = 0; e < kFinB; ++e) os[e][i] = e < nb ? __ldcg(a.orot + (((size_t)lc * B + b0 + e) * H + h) * D + i) : 0.f;
  __syncthreads();
  // the same summation order as the fused epilogue of decode_main_kernel (32-element chunks, four interleaved chains),
  // so that both forms give identical bits
  float acc[kFinB];
#pragma unroll
  for (int e = 0; e < kFinB; ++e) acc[e] = 0.f;
#pragma unroll 1
  for (int k0 = 0; k0 < D; k0 += 32) {
    if (k0 > 0) {
#pragma unroll
      for (int k = 0; k < 32; ++k) pv[k] = __ldg(Pv + (size_t)(k0 + k) * D + i);
    }
#pragma unroll
    for (int e = 0; e < kFinB; ++e) {
      float r0 = 0.f, r1 = 0.f, r2 = 0.f, r3 = 0.f;
#pragma unroll
      for (int k = 0; k < 32; k += 4) {
        r0 = fmaf(pv[k], os[e][k0 + k], r0);
        r1 = fmaf(pv[k + 1], os[e][k0 + k + 1], r1);
        r2 = fmaf(pv[k + 2], os[e][k0 + k + 2], r2);
        r3 = fmaf(pv[k + 3], os[e][k0 + k + 3], r3);
      }
      acc[e] += (r0 + r1) + (r2 + r3);
    }
  }
  for (int e = 0; e < nb; ++e) {
    TIO* outp = reinterpret_cast<TIO*>(a.out) + (((size_t)lc * B + b0 + e) * H + h) * D;
    if constexpr (sizeof(TIO) == 2) outp[i] = __float2half_rn(acc[e]);
    else outp[i] = acc[e];
  }
}

// ------------------------------------------------------------------------------------------ launchers
template <int D, typename T, bool kFusedOut, bool kVq>
static cudaError_t launch_decode_t(const DecodeArgs& a, cudaStream_t st) {
  constexpr int smem = DecodeCfg<D, kVq>::kSmemBytes;
  // per launch: the attribute is per device and a process may drive several
  cudaError_t e = cudaFuncSetAttribute(decode_main_kernel<D, T, kFusedOut, kVq>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(a.nsplit, a.cv.H, a.n_layers_call * a.cv.B);
  cfg.blockDim = dim3(kDecodeThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  e = cudaLaunchKernelEx(&cfg, decode_main_kernel<D, T, kFusedOut, kVq>, a);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

template <int D, typename T>
static cudaError_t launch_finish_t(const DecodeArgs& a, bool programmatic, cudaStream_t st) {
  const int nbg = (a.cv.B + kFinB - 1) / kFinB;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(a.n_layers_call * a.cv.H * nbg);
  cfg.blockDim = dim3(D);
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = programmatic ? 1 : 0;  // after a kernel of the same stream only (the stepper puts it behind a copy)
  cudaError_t e = cudaLaunchKernelEx(&cfg, finish_kernel<D, T>, a, nbg);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_finish(const DecodeArgs& a, int D, bool programmatic, cudaStream_t st) {
  if (D == 64) return a.dt == TQ_F16 ? launch_finish_t<64, __half>(a, programmatic, st) : launch_finish_t<64, float>(a, programmatic, st);
  return a.dt == TQ_F16 ? launch_finish_t<128, __half>(a, programmatic, st) : launch_finish_t<128, float>(a, programmatic, st);
}

int decode_ctas_per_sm(int D) { return D == 64 ? DecodeCfg<64>::kCtasPerSm : DecodeCfg<128>::kCtasPerSm; }

template <bool kVq>
static cudaError_t launch_decode_v(const DecodeArgs& a, int D, bool fused_out, cudaStream_t st) {
  if (fused_out) {
    if (D == 64) return a.dt == TQ_F16 ? launch_decode_t<64, __half, true, kVq>(a, st) : launch_decode_t<64, float, true, kVq>(a, st);
    return a.dt == TQ_F16 ? launch_decode_t<128, __half, true, kVq>(a, st) : launch_decode_t<128, float, true, kVq>(a, st);
  }
  if (D == 64) return launch_decode_t<64, __half, false, kVq>(a, st);  // the output type is finish_kernel's business
  return launch_decode_t<128, __half, false, kVq>(a, st);
}

cudaError_t launch_decode(const DecodeArgs& a, int D, bool fused_out, cudaStream_t st) {
  return a.cv.vsk ? launch_decode_v<true>(a, D, fused_out, st) : launch_decode_v<false>(a, D, fused_out, st);
}

int decode_record_floats(int D, bool vq) { return vq ? 2 * D + 3 : D + 2; }

}  // namespace tq
