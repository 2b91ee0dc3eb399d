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
// Split-K over the sequence: grid = units x nsplit CTAs (nsplit chosen on the host from t_hint so that the SMs
// carry equal work); a unit covered by one CTA is finished in place, otherwise the last CTA to arrive merges
// the partial (m, l, o') triples.  Either way the finishing CTA applies PI_V^T.
// Tokens whose softmax weight underflows to exactly 0 in fp32 add nothing to o': their V lookups are skipped
// (a warp-uniform test on a ballot of the weights), which changes no bit of the result.
#include <utility>

#include "tq_common.cuh"

namespace tq {


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

constexpr int kMaxSegments = 64;      // split-K partial slots per unit (tq_api.cu sizes the workspace)
#ifndef TQ_DECODE_CTAS64
#define TQ_DECODE_CTAS64 5
#endif
#ifndef TQ_DECODE_THREADS
#define TQ_DECODE_THREADS 128
#endif
constexpr int kDecodeThreads = TQ_DECODE_THREADS;  // warps of one CTA share the tables of one unit
constexpr int kDecodeWarps = kDecodeThreads / 32;
constexpr int kBuildThreads = 128;  // threads that build the tables and apply PI_V^T

// Shared-memory map in ABSOLUTE shared-window addresses (the OR-addressing needs the K/V tables aligned to
// their own size, the sign table to 4 KB).  Dynamic shared memory starts right after the 1 KB the driver
// reserves, so everything is placed at fixed absolute addresses and the kernel traps if the window starts
// later than kAbsWbuf.
template <int D>
struct DecodeCfg {
  using Lo = Layout<D>;
  static constexpr int NCK = D;                          // columns of the K table = 2 P (>= P + 31)
  static constexpr int LSK = D == 64 ? 8 : 9;            // log2(NCK * 4)
  static constexpr int kKtabBytes = 64 * NCK * 4;        // 16 KB | 32 KB
  static constexpr int kVtabBytes = 64 * 16 * 8;         // 8 KB: [entry][lane mod 16] float2 (64-bit reads are
                                                         // served one half-warp at a time)
  static constexpr int kStabBytes = 16 * 64 * 4;         // 4 KB
  static constexpr unsigned kAbsWbuf = 2048;             // 4 warps x 32 softmax weights, then the arrival flag
  static constexpr unsigned kAbsStab = 4096;
  static constexpr unsigned kAbsVtab = 8192;
  static constexpr unsigned kAbsKtab = D == 64 ? 16384 : 32768;
  static constexpr unsigned kAbsScratch = D == 64 ? 32768 : 16384;  // per-warp partials, merged o
  static constexpr int kScratchBytes = 16 + 8 * (D + 2) * 4 + 2 * D * 4;  // up to 8 warps
  static constexpr unsigned kAbsEnd = D == 64 ? kAbsScratch + kScratchBytes : kAbsKtab + kKtabBytes;
  static constexpr int kSmemBytes = kAbsEnd;             // requested dynamic bytes (window start <= 2 KB)
  static constexpr int kCtasPerSm = D == 64 ? TQ_DECODE_CTAS64 : 3;
};

// ---- packed fp32x2 arithmetic (sm_100: FFMA2 / FADD2 / FMUL2 issue two fp32 operations per slot) ----------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 lds_b64(unsigned addr) {
  f32x2 v;
  asm("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
  return v;
}

// <q'', lut_K[codes]>: P table reads, summed two at a time
// pairwise (tree) sum of N packed pairs, then of the two halves: short dependency chains for the scheduler
template <int N>
__device__ __forceinline__ float tree_sum(f32x2 (&v)[N]) {
#pragma unroll
  for (int n = N / 2; n >= 1; n >>= 1)
#pragma unroll
    for (int i = 0; i < n; ++i) v[i] = add2(v[i], v[i + n]);
  float a, b;
  unpack2(v[0], a, b);
  return a + b;
}
template <int D, int... K>
__device__ __forceinline__ float k_score(const unsigned (&kw)[Layout<D>::KCW], unsigned kbase,
                                         std::integer_sequence<int, K...>) {
  // all table addresses first, then all reads, then the sum: three wide phases instead of 32 short chains
  const unsigned a0[sizeof...(K)] = {(field_at<DecodeCfg<D>::LSK, 12 * K, 6>(kw) | kbase)...};
  const unsigned a1[sizeof...(K)] = {(field_at<DecodeCfg<D>::LSK, 12 * K + 6, 6>(kw) | kbase)...};
  f32x2 v[sizeof...(K)] = {pack2(lds_f32<8 * K>(a0[K]), lds_f32<8 * K + 4>(a1[K]))...};
  return tree_sum(v);
}

// <z, sigma>: d/4 nibble-table reads
template <int D, int... K>
__device__ __forceinline__ float s_score(const unsigned (&sw)[Layout<D>::KSW], unsigned sbase,
                                         std::integer_sequence<int, K...>) {
  const unsigned a0[sizeof...(K)] = {(field_at<8, 8 * K, 4>(sw) | sbase)...};
  const unsigned a1[sizeof...(K)] = {(field_at<8, 8 * K + 4, 4>(sw) | sbase)...};
  f32x2 v[sizeof...(K)] = {pack2(lds_f32<8 * K>(a0[K]), lds_f32<8 * K + 4>(a1[K]))...};
  return tree_sum(v);
}

// V accumulate, lane = coordinate pair: for token J of the tile, o2[part] += w_J * (lut_V[c0], lut_V[c1])
template <int D, int J>
__device__ __forceinline__ void v_token(const unsigned (&vw)[Layout<D>::KCW], unsigned vbase, float w,
                                        f32x2 (&o2)[2 * (Layout<D>::P / kTile)]) {
  const f32x2 w2 = pack2(w, w);
#pragma unroll
  for (int part = 0; part < Layout<D>::P / kTile; ++part) {
    unsigned f = part == 0 ? field_at<7, 6 * J, 6>(vw) : field_at<7, 192 * (Layout<D>::P / kTile - 1) + 6 * J, 6>(vw);
    o2[2 * part + (J & 1)] = fma2(lds_b64(f | vbase), w2, o2[2 * part + (J & 1)]);
  }
}
template <int D, int... J>
__device__ __forceinline__ void v_accum(const unsigned (&vw)[Layout<D>::KCW], unsigned vbase, unsigned wbuf,
                                        unsigned nz /* ballot: token slots with a non-zero weight */,
                                        f32x2 (&o2)[2 * (Layout<D>::P / kTile)], std::integer_sequence<int, J...>) {
  // w of tokens 4J .. 4J+3 arrive with one broadcast 128-bit read; groups whose weights are all 0 are skipped
  (([&] {
     if (nz & (0xfu << (4 * J))) {
       float4 w4;
       asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];"
                    : "=f"(w4.x), "=f"(w4.y), "=f"(w4.z), "=f"(w4.w)
                    : "r"(wbuf), "n"(16 * J));
       v_token<D, 4 * J>(vw, vbase, w4.x, o2);
       v_token<D, 4 * J + 1>(vw, vbase, w4.y, o2);
       v_token<D, 4 * J + 2>(vw, vbase, w4.z, o2);
       v_token<D, 4 * J + 3>(vw, vbase, w4.w, o2);
     }
   }()),
   ...);
}

// What one lane loads per tile: its own token's K code / sign strings and norms (lane = token), and the V
// code string of its coordinate pair(s) for all 32 tokens (lane = pair).
template <int D>
struct TileWords {
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
__device__ __forceinline__ void load_tile_words(TileWords<D>& t, const unsigned char* tp, int lane) {
  using Lo = Layout<D>;
  load_words<Lo::KCW>(t.kw, tp + Lo::kOffKC, lane);
  load_words<Lo::KSW>(t.sw, tp + Lo::kOffKS, lane);
  load_words<Lo::KCW>(t.vw, tp + Lo::kOffVC, lane);
  t.kn = __ldg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffKN) + lane);
  t.kr = __ldg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffKR) + lane);
  t.vn = __ldg(reinterpret_cast<const unsigned short*>(tp + Lo::kOffVN) + lane);
}

// ---- table construction (per CTA; the prep kernel stores q'' and z pre-scaled so that logits come out in
//      log2 units: q'' * log2(e)/sqrt(d), z * log2(e)/sqrt(d) * sqrt(pi/2)/m) ------------------------------------
// Every thread owns four consecutive table columns and writes them with 128-bit stores.
template <int D>
struct TableInputs {  // everything a thread needs from global memory, requested before anything is used
  float4 qa[1], qb[1];
  float4 zz[4];
  float4 lk0, lk1, lv0, lv1;
};

template <int D>
__device__ __forceinline__ void load_table_inputs(TableInputs<D>& t, const float* qr, const float* __restrict__ lk,
                                                  const float* __restrict__ lv, int tid) {
  using Lo = Layout<D>;
  using Cfg = DecodeCfg<D>;
  constexpr int NQ = Cfg::NCK / 4;
  const int g0 = (4 * (tid % NQ)) % Lo::P;
  t.qa[0] = __ldcg(reinterpret_cast<const float4*>(qr + 2 * g0));
  t.qb[0] = __ldcg(reinterpret_cast<const float4*>(qr + 2 * g0) + 1);
  const int n0 = (4 * (tid % 16)) % Lo::NG;
#pragma unroll
  for (int i = 0; i < 4; ++i) t.zz[i] = __ldcg(reinterpret_cast<const float4*>(qr + D + 4 * (n0 + i)));
  t.lk0 = __ldg(reinterpret_cast<const float4*>(lk));
  t.lk1 = __ldg(reinterpret_cast<const float4*>(lk) + 1);
  t.lv0 = __ldg(reinterpret_cast<const float4*>(lv));
  t.lv1 = __ldg(reinterpret_cast<const float4*>(lv) + 1);
}

template <int D>
__device__ __forceinline__ void build_tables(float* Ktab, float* Stab, float2* Vtab, const TableInputs<D>& t, int tid) {
  using Lo = Layout<D>;
  using Cfg = DecodeCfg<D>;
  const float lut[8] = {t.lk0.x, t.lk0.y, t.lk0.z, t.lk0.w, t.lk1.x, t.lk1.y, t.lk1.z, t.lk1.w};
  {  // Ktab[8 hi + lo][c] = q''_{2g} lut[lo] + q''_{2g+1} lut[hi],  g = c mod P
    constexpr int NQ = Cfg::NCK / 4;                // column quads: 16 | 32
    constexpr int HPT = 8 / (kBuildThreads / NQ);  // hi codes per thread: 1 | 2
    const int cq = tid % NQ, eg = tid / NQ;
    const float q0[4] = {t.qa[0].x, t.qa[0].z, t.qb[0].x, t.qb[0].z};  // q''_{2g}
    const float q1[4] = {t.qa[0].y, t.qa[0].w, t.qb[0].y, t.qb[0].w};  // q''_{2g+1}
#pragma unroll
    for (int hh = 0; hh < HPT; ++hh) {
      const int hi = eg * HPT + hh;
      float lh = lut[0];
#pragma unroll
      for (int c = 1; c < 8; ++c) lh = (hi == c) ? lut[c] : lh;
      const float b0 = q1[0] * lh, b1 = q1[1] * lh, b2 = q1[2] * lh, b3 = q1[3] * lh;
      float* dst = Ktab + (size_t)(hi * 8) * Cfg::NCK + 4 * cq;
#pragma unroll
      for (int lo = 0; lo < 8; ++lo)
        *reinterpret_cast<float4*>(dst + lo * Cfg::NCK) =
            make_float4(fmaf(q0[0], lut[lo], b0), fmaf(q0[1], lut[lo], b1), fmaf(q0[2], lut[lo], b2), fmaf(q0[3], lut[lo], b3));
    }
  }
  {  // Stab[e][c] = sum_b (bit b of e ? +z : -z)[4n + b],  n = c mod NG; 16 column quads x 8 entry pairs
    const int cq = tid % 16, eg = tid / 16;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int e = 2 * eg + j;
      const float s0 = (e & 1) ? 1.f : -1.f, s1 = (e & 2) ? 1.f : -1.f, s2 = (e & 4) ? 1.f : -1.f, s3 = (e & 8) ? 1.f : -1.f;
      float v[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) v[i] = fmaf(s0, t.zz[i].x, fmaf(s1, t.zz[i].y, fmaf(s2, t.zz[i].z, s3 * t.zz[i].w)));
      *reinterpret_cast<float4*>(Stab + e * 64 + 4 * cq) = make_float4(v[0], v[1], v[2], v[3]);
    }
  }
  {  // Vtab[8 hi + lo][col] = (lut_V[lo], lut_V[hi]); 128 threads: hi = tid / 16, col = tid % 16
    const float lv[8] = {t.lv0.x, t.lv0.y, t.lv0.z, t.lv0.w, t.lv1.x, t.lv1.y, t.lv1.z, t.lv1.w};
    const int col = tid & 15, eq = tid >> 4;
    float hi = lv[0];
#pragma unroll
    for (int c = 1; c < 8; ++c) hi = (eq == c) ? lv[c] : hi;
#pragma unroll
    for (int j = 0; j < 8; ++j) Vtab[(eq * 8 + j) * 16 + col] = make_float2(lv[j], hi);
  }
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

// ---- the streaming kernel ------------------------------------------------------------------------------------
// grid = units x nsplit.  CTA (unit uc, split sp) streams tiles [sp * per, (sp + 1) * per) of its unit, where
// per = ceil(ceil(T / 32) / nsplit) is derived on the device from seq_len, so a shorter cache simply leaves the
// trailing splits empty.  The four warps take tiles round-robin with a register double buffer.
template <int D, typename TIO>
__global__ void __launch_bounds__(kDecodeThreads, DecodeCfg<D>::kCtasPerSm) decode_main_kernel(DecodeArgs a) {
  using Lo = Layout<D>;
  using Cfg = DecodeCfg<D>;
  constexpr int NW = kDecodeWarps;
  constexpr int VP = Lo::P / kTile;  // coordinate pairs per lane: 1 | 2
  extern __shared__ unsigned char smem_raw[];
  const unsigned raw = (unsigned)__cvta_generic_to_shared(smem_raw);
  if (raw > Cfg::kAbsWbuf) __trap();  // the fixed shared-memory map does not fit: fail loudly
  unsigned char* abs0 = smem_raw - raw;  // generic pointer to absolute shared address 0 of this CTA's window
  float* Stab = reinterpret_cast<float*>(abs0 + Cfg::kAbsStab);
  float* red = reinterpret_cast<float*>(abs0 + Cfg::kAbsScratch + 16);  // NW x (D + 2)
  float* omerged = red + NW * (D + 2);                                   // [D] + [D] partial matvec
  float* wbuf_f = reinterpret_cast<float*>(abs0 + Cfg::kAbsWbuf);       // NW x 32 softmax weights
  int* flag = reinterpret_cast<int*>(wbuf_f + NW * 32);
  float* Ktab = reinterpret_cast<float*>(abs0 + Cfg::kAbsKtab);
  float2* Vtab = reinterpret_cast<float2*>(abs0 + Cfg::kAbsVtab);
  const unsigned ktab = Cfg::kAbsKtab, vtab = Cfg::kAbsVtab, stab = Cfg::kAbsStab;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int B = a.cv.B, H = a.cv.H;
  const int nsplit = a.nsplit;
  const int uc = (int)blockIdx.x / nsplit, sp = (int)blockIdx.x - uc * nsplit;
  const int e = uc / H, h = uc - e * H;  // e = (layer-in-call, batch); seq_len is contiguous over e
  const int lc = e / B, b = e - lc * B;
  const int layer = a.layer_begin + lc;
  const size_t lh = (size_t)layer * H + h;
  {  // before the PDL wait: hints only.  The cache stream of this CTA starts towards L2 while the prep kernel in front
     // of this launch is still running (it rewrites at most one tile per unit, and L2 stays coherent); PI_V too.
    const int per0 = a.per, t0 = sp * per0;
    const int c1 = sp == nsplit - 1 ? a.cv.tiles_cap : min(a.cv.tiles_cap, t0 + per0);
    const unsigned char* st0 = a.cv.tiles + (((size_t)layer * B + b) * H + h) * a.cv.stream_bytes;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const int t = t0 + warp + i * NW;
      if (t < c1 && lane == 0)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(st0 + (size_t)t * Lo::kTileBytes), "r"(Lo::kTileBytes)
                     : "memory");
    }
  }
  pdl_wait();
  // ---- every global request the prologue depends on goes out first and together: the cache length, the table
  //      inputs, then (speculatively, from the host's split plan) this warp's first tile, so that the small loads
  //      never queue behind the bulk ones
  int T;
  asm volatile("ld.global.b32 %0, [%1];" : "=r"(T) : "l"(a.cv.seq_len + a.layer_begin * B + e));
  TableInputs<D> tin;
  if (tid < kBuildThreads) load_table_inputs<D>(tin, a.qrot + (size_t)uc * 2 * D, a.lut_k + lh * 8, a.lut_v + lh * 8, tid);
  const int per = a.per;  // tiles per split planned from t_hint; the last split also takes whatever lies beyond
  const int tile0 = sp * per;
  const int cap1 = sp == nsplit - 1 ? a.cv.tiles_cap : min(a.cv.tiles_cap, tile0 + per);  // static bound of this split
  const unsigned char* stream = a.cv.tiles + (((size_t)layer * B + b) * H + h) * a.cv.stream_bytes;
  TileWords<D> bufA, bufB;  // register double buffer, ping-pong (no copies)
  if (tile0 + warp < cap1) load_tile_words<D>(bufA, stream + (size_t)(tile0 + warp) * Lo::kTileBytes, lane);
  auto prefetch_tile = [&](int t, int bound) {  // one bulk L2 prefetch per tile, issued by one lane
    if (t < bound && lane == 0)
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(stream + (size_t)t * Lo::kTileBytes),
                   "r"(Lo::kTileBytes)
                   : "memory");
  };
  constexpr int kPrefetchAhead = 3;  // rounds of NW tiles
  const float* Pv = a.pi_v + lh * D * D;
#pragma unroll
  for (int i = 0; i < D * D * 4 / 128 / kBuildThreads; ++i)
    if (tid < kBuildThreads) asm volatile("prefetch.global.L2 [%0];" ::"l"(Pv + (size_t)(i * kBuildThreads + tid) * 32));
  const int nt = (T + kTile - 1) / kTile;
  if (tile0 >= nt) return;  // empty cache (the prep kernel wrote out = 0) or a trailing split with nothing to do
  const int tile1 = min(nt, cap1);
  const int nseg = min(nsplit, (nt + per - 1) / per);  // splits of this unit that have work
  if (tid < kBuildThreads) build_tables<D>(Ktab, Stab, Vtab, tin, tid);
  __syncthreads();

  // table base | lane column as ONE register.  ptxas sees through an empty asm and would split the constant base
  // from the lane term again (an extra LOP3 per lookup); XOR with a kernel argument that is always 0 keeps it whole,
  // so every lookup address is a single LOP3: (field & mask) | base.
  const unsigned kbase = (ktab + lane * 4) ^ (unsigned)a.zero, sbase = (stab + lane * 4) ^ (unsigned)a.zero,
                 vbase = (vtab + (lane & 15) * 8) ^ (unsigned)a.zero;
  const unsigned wbuf = (unsigned)__cvta_generic_to_shared(wbuf_f + warp * 32);

  f32x2 o2[2 * VP];  // [pair][even / odd tokens]
#pragma unroll
  for (int i = 0; i < 2 * VP; ++i) o2[i] = 0ull;
  float m = -INFINITY, l = 0.f;

  // one 32-token tile: scores (lane = token) -> online softmax -> V accumulate (lane = coordinate pair)
  auto process = [&](const TileWords<D>& tw, int tile) {
    const bool valid = tile * kTile + lane < T;
    const float sa = k_score<D>(tw.kw, kbase, std::make_integer_sequence<int, Lo::P / 2>{});
    const float sb = s_score<D>(tw.sw, sbase, std::make_integer_sequence<int, Lo::NG / 2>{});
    float s2 = f16_bits_to_f32(tw.kn) * fmaf(f16_bits_to_f32(tw.kr), sb, sa);
    s2 = valid ? s2 : -INFINITY;
    const float mnew = fmaxf(m, warp_max_f32(s2));  // finite: slot 0 of every processed tile is valid
    const float fsc = ex2_ftz(m - mnew);            // 0 on a warp's first tile (m = -inf)
    m = mnew;
    const float p = ex2_ftz(s2 - m);                // invalid lanes: exp2(-inf) = 0
    l = fmaf(l, fsc, p);
    const f32x2 fsc2 = pack2(fsc, fsc);
#pragma unroll
    for (int i = 0; i < 2 * VP; ++i) o2[i] = mul2(o2[i], fsc2);
    const float wv = valid ? p * f16_bits_to_f32(tw.vn) : 0.f;
    const unsigned nz = __ballot_sync(0xffffffffu, wv != 0.f);
    if (nz) {
      // hand the softmax weights from lane = token to lane = coordinate pair through shared memory
      __syncwarp();
      asm volatile("st.shared.f32 [%0], %1;" ::"r"(wbuf + lane * 4), "f"(wv));
      __syncwarp();
      v_accum<D>(tw.vw, vbase, wbuf, nz, o2, std::make_integer_sequence<int, kTile / 4>{});
    }
  };
  auto fetch = [&](TileWords<D>& tw, int tile) {
    prefetch_tile(tile + (kPrefetchAhead - 1) * NW, tile1);
    if (tile < tile1) load_tile_words<D>(tw, stream + (size_t)tile * Lo::kTileBytes, lane);
  };
  int tile = tile0 + warp;
  while (tile < tile1) {
    fetch(bufB, tile + NW);
    process(bufA, tile);
    tile += NW;
    if (tile >= tile1) break;
    fetch(bufA, tile + NW);
    process(bufB, tile);
    tile += NW;
  }

  // ---- reduce over the CTA's warps (lanes already own distinct coordinates)
  l = warp_sum(l);
  float* wr = red + warp * (D + 2);
  if (lane == 0) {
    wr[0] = m;
    wr[1] = l;
  }
#pragma unroll
  for (int i = 0; i < VP; ++i) {
    float x0, x1;
    unpack2(add2(o2[2 * i], o2[2 * i + 1]), x0, x1);
    wr[2 + 2 * (lane + kTile * i)] = x0;
    wr[2 + 2 * (lane + kTile * i) + 1] = x1;
  }
  __syncthreads();
  float M = -INFINITY;
#pragma unroll
  for (int w = 0; w < NW; ++w) M = fmaxf(M, red[w * (D + 2)]);
  float Lsum = 0.f, oi = 0.f;
  if (tid < D) {
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const float mw = red[w * (D + 2)];
      const float fw = mw == -INFINITY ? 0.f : ex2_ftz(mw - M);
      Lsum = fmaf(red[w * (D + 2) + 1], fw, Lsum);
      oi = fmaf(red[w * (D + 2) + 2 + tid], fw, oi);
    }
  }
  if (nseg > 1) {
    float* part = a.partials + ((size_t)uc * kMaxSegments + sp) * (D + 2);
    if (tid < D) part[2 + tid] = oi;
    if (tid == 0) {
      part[0] = M;
      part[1] = Lsum;
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
    if (*flag == 0) return;
    const float* pp = a.partials + (size_t)uc * kMaxSegments * (D + 2);
    M = -INFINITY;
    for (int s = 0; s < nseg; ++s) M = fmaxf(M, __ldcg(pp + s * (D + 2)));
    Lsum = 0.f;
    oi = 0.f;
    if (tid < D) {
      for (int s = 0; s < nseg; ++s) {
        const float ms = __ldcg(pp + s * (D + 2));
        const float fs = ms == -INFINITY ? 0.f : ex2_ftz(ms - M);
        Lsum = fmaf(__ldcg(pp + s * (D + 2) + 1), fs, Lsum);
        oi = fmaf(__ldcg(pp + s * (D + 2) + 2 + tid), fs, oi);
      }
    }
  }
  // ---- out = PI_V^T (o' / l): the k range is split over the 128 / D thread groups
  if (tid < D) omerged[tid] = Lsum > 0.f ? oi / Lsum : 0.f;
  __syncthreads();
  constexpr int PARTS = kBuildThreads / D;  // 2 | 1
  constexpr int KP = D / PARTS;             // 32 | 128
  const int i = tid % D, part = (tid / D) % PARTS;
  float r = 0.f;
  if (tid < kBuildThreads) {
    const float* Pvp = Pv + (size_t)part * KP * D + i;
#pragma unroll 32
    for (int k = 0; k < KP; ++k) r = fmaf(__ldg(Pvp + (size_t)k * D), omerged[part * KP + k], r);
  }
  if (PARTS > 1 && tid < kBuildThreads && part > 0) omerged[part * D + i] = r;
  __syncthreads();
  if (tid < D) {
#pragma unroll
    for (int pp = 1; pp < PARTS; ++pp) r += omerged[pp * D + i];
    TIO* outp = reinterpret_cast<TIO*>(a.out) + (size_t)uc * D;
    if constexpr (sizeof(TIO) == 2) outp[i] = __float2half_rn(r);
    else outp[i] = r;
  }
}

// ------------------------------------------------------------------------------------------ launchers
template <int D, typename T>
static cudaError_t launch_decode_t(const DecodeArgs& a, cudaStream_t st) {
  cudaError_t e;
  constexpr int smem = DecodeCfg<D>::kSmemBytes;
  static bool attr_set = false;
  if (!attr_set) {
    e = cudaFuncSetAttribute(decode_main_kernel<D, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int units = a.n_layers_call * a.cv.B * a.cv.H;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(units * a.nsplit);
  cfg.blockDim = dim3(kDecodeThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = a.nsplit == 1 ? 1 : 0;  // measured: early scheduling helps one-CTA-per-unit launches, hurts split ones
  e = cudaLaunchKernelEx(&cfg, decode_main_kernel<D, T>, a);
  count_launch();
  return e != cudaSuccess ? e : cudaGetLastError();
}

int decode_ctas_per_sm(int D) { return D == 64 ? DecodeCfg<64>::kCtasPerSm : DecodeCfg<128>::kCtasPerSm; }

cudaError_t launch_decode(const DecodeArgs& a, int D, cudaStream_t st) {
  if (D == 64) return a.dt == TQ_F16 ? launch_decode_t<64, __half>(a, st) : launch_decode_t<64, float>(a, st);
  return a.dt == TQ_F16 ? launch_decode_t<128, __half>(a, st) : launch_decode_t<128, float>(a, st);
}

}  // namespace tq
