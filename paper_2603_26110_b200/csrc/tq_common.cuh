// tq_common.cuh — shared device/host definitions of the CUDA product path (sm_100a).
// Device cache layout as documented in include/tq.h ("Device cache format").  Nothing here is shared with
// oracle/.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tq.h"

namespace tq {

constexpr int kTile = TQ_TILE_TOKENS;  // tokens per tile == lanes per warp

// ---- per-head-dim tile layout ------------------------------------------------------------------------
// The fused decode kernel runs its three contractions (<q'', lut_K[codes]>, <z, sigma>, sum_j w_j lut_V[codes_j]) as
// warp-level mma.sync.m16n8k16 with fp16 operands built in registers, so a tile of 32 tokens is stored in exactly the
// order of the m16n8k16 A-fragment: lane = 4 g + t (g = lane / 4 = fragment row, t = lane % 4 = fragment column group).
//   K codes : lane (g, t) owns, for the four token slots s = g + 8 r (r = 0..3), the six-bit pair fields
//             (code_{2p} | code_{2p+1} << 3) of the pairs p = t + 4 j (j < J = d/8); field (r, j) sits at bit
//             6 (J r + j) of the lane's string of KCW = 3d/32 words;
//   K signs : lane (g, t) owns sketch rows [t d/4, (t+1) d/4) of the same four slots, as 16-bit pieces u < d/64;
//             the pieces of slots g + 16 mt ("A") and g + 8 + 16 mt ("B") are byte-interleaved in word (mt, u):
//             bytes [A bits 0..7 | B bits 0..7 | A bits 8..15 | B bits 8..15], so that (word >> 8 ab) & (0x00010001 << p)
//             is an fp16x2 register holding two sign bits as the (subnormal) values 2^(p-24);
//   V codes : lane (g, t) owns coordinates i = g + 8 c (c < C = d/8) of the token pairs pp = t + 4 j (j < 4); field
//             (j, c) = code_i(token 2pp) | code_i(token 2pp+1) << 3 sits at bit 6 (C j + c);
//   norms   : lane (g, t) owns token slot g + 8 t: one u32 (|k| | |r_k| << 16, binary16 bits) and one u16 (|v|).
// A "section" is a per-lane string of W 32-bit words stored chunk-major: 16-byte chunks [c][lane], then (if
// W % 4 == 2) one 8-byte chunk [lane].  62 (d = 64) / 118 (d = 128) bytes per token, as the canonical format.
template <int D>
struct Layout {
  static_assert(D == 64 || D == 128, "head_dim must be 64 or 128");
  static constexpr int P = D / 2;            // coordinate pairs per vector
  static constexpr int J = D / 8;            // K pair fields per (lane, token slot)
  static constexpr int C = D / 8;            // V coordinates per lane
  static constexpr int U = D / 64;           // 16-bit sign pieces per (lane, token slot)
  static constexpr int KCW = 3 * D / 32;     // words per lane of the K (or V) code section: 6 | 12
  static constexpr int KSW = D / 32;         // words per lane of the sign section: 2 | 4
  static constexpr int kCodeBytes = KCW * 4 * kTile;
  static constexpr int kSignBytes = KSW * 4 * kTile;
  static constexpr int kOffKC = 0;
  static constexpr int kOffKS = kOffKC + kCodeBytes;
  static constexpr int kOffVC = kOffKS + kSignBytes;
  static constexpr int kOffNK = kOffVC + kCodeBytes;  // u32 per lane: binary16 |k| | binary16 |r_k| << 16
  static constexpr int kOffVN = kOffNK + 4 * kTile;   // u16 per lane: binary16 |v|
  static constexpr int kTileBytes = kOffVN + 2 * kTile;  // 1984 | 3776
  static constexpr int kBytesPerToken = kTileBytes / kTile;
};

// byte offset (inside its section) of word w of lane l, section of W words per lane
__host__ __device__ constexpr int word_offset(int W, int w, int l) {
  return (w < (W / 4) * 4) ? ((w / 4) * 16 * kTile + l * 16 + (w % 4) * 4)
                           : ((W / 4) * 16 * kTile + l * 8 + (w - (W / 4) * 4) * 4);
}

// lane that owns token slot s for the norms and the softmax, and its inverse
__host__ __device__ constexpr int slot_lane(int s) { return 4 * (s & 7) + (s >> 3); }
__host__ __device__ constexpr int lane_slot(int l) { return (l >> 2) + 8 * (l & 3); }

struct BitPos {
  int lane, bit;  // bit offset inside the lane's word string of that section
};
// six-bit K pair field of (slot s, pair p)
template <int D>
__host__ __device__ constexpr BitPos k_field_pos(int s, int p) {
  return BitPos{4 * (s & 7) + (p & 3), 6 * (Layout<D>::J * (s >> 3) + (p >> 2))};
}
// sign bit of (slot s, sketch row rho)
template <int D>
__host__ __device__ constexpr BitPos sign_bit_pos(int s, int rho) {
  const int t = rho / (D / 4), i = rho % (D / 4), u = i >> 4, ib = i & 15;
  const int word = (s >> 4) * Layout<D>::U + u, byte = (ib >> 3) * 2 + ((s >> 3) & 1);
  return BitPos{4 * (s & 7) + t, 32 * word + 8 * byte + (ib & 7)};
}
// three-bit V code of (slot s, coordinate i)
template <int D>
__host__ __device__ constexpr BitPos v_code_pos(int s, int i) {
  const int pp = s >> 1;
  return BitPos{4 * (i & 7) + (pp & 3), 6 * (Layout<D>::C * (pp >> 2) + (i >> 3)) + 3 * (s & 1)};
}

// ---- V-side sketch tiles (tq_shape.v_qjl = 1; Algorithm 1 line 10) ------------------------------------------
// A second stream of tiles per unit, one per 32 tokens, next to the main stream (which stays exactly as above):
//   V signs : KSW words per lane in the A-fragment order of  b[rho] += bits^T (16 sketch rows x 16 tokens) x w' :
//             sketch row rho = 16 mt + 8 rh + g, token slot s = 16 ks + 8 th + 2 t + e  ->  lane (g, t),
//             word ks (D/64) + (mt >> 2), bit 16 e + 4 (mt & 3) + 2 rh + th, so that word & (0x00010001 << p) is an
//             fp16 pair (token 2t [+8 th], token 2t + 1 [+8 th]) of one sketch row with halves 0 or 2^(p - 24);
//   v_rnorm : one u16 per lane (binary16 |r_v|), lane (g, t) owns slot g + 8 t as for the other norms.
// 10 (d = 64) / 18 (d = 128) bytes per token.
template <int D>
struct VskLayout {
  static constexpr int KSW = D / 32;
  static constexpr int kSignBytes = KSW * 4 * kTile;
  static constexpr int kOffVS = 0;
  static constexpr int kOffVR = kSignBytes;
  static constexpr int kTileBytes = kSignBytes + 2 * kTile;  // 320 | 576
};
template <int D>
__host__ __device__ constexpr BitPos vsign_bit_pos(int s, int rho) {
  const int ks = s >> 4, th = (s >> 3) & 1, t = (s & 7) >> 1, e = s & 1;
  const int mt = rho >> 4, rh = (rho >> 3) & 1, g = rho & 7;
  return BitPos{4 * g + t, 32 * (ks * (D / 64) + (mt >> 2)) + 16 * e + 4 * (mt & 3) + 2 * rh + th};
}

// ---- per-unit operands of the fused decode kernel (written by the prep kernel into the workspace) -------------------
// The decode kernel feeds q'' and z to mma.sync.m16n8k16 as B fragments in fp16, split hi + lo (column n of B holds
// the hi part for even n and the lo part for odd n).  A lane (g, t) needs the pattern x = g & 1, t:
//   words [0, 2 KS)    bq[ks][reg] : q''_s (16 ks + 2 t + 8 reg), (.. + 1)           q''_s = q'' log2(e)/sqrt(d) 2^eq
//   words [2 KS, 4 KS) bz[ks][reg] : z_s (rho), z_s (rho + 8), rho = t d/4 + 16 (ks / 4) + 2 (ks % 4) + reg,
//                                    scaled by 2^(ez - 2 (ks % 4) - reg)             z_s = z log2(e)/sqrt(d) sqrt(pi/2)/m
// followed by four floats: kscale = 2^-eq, sscale = 2^(25 - ez), zsum = sum_rho z_s(rho), 0.
template <int D>
struct FragLayout {
  static constexpr int KS = D / 16;
  static constexpr int kWordsPerPat = 4 * KS;               // 16 | 32
  static constexpr int kScalOff = 8 * kWordsPerPat;         // in words
  static constexpr int kWords = kScalOff + 4;
  static constexpr int kBytes = kWords * 4;                 // 528 | 1040
};
// Dequantisation tables of one (layer, head), also written by the prep kernel: [K hi | K lo | V hi | V lo][64] fp16
// pairs (entry c0 | c1 << 3 -> (lut[c0], lut[c1]), lo = lut - hi), then one word: 1 if every lo is zero.
constexpr int kTabWords = 4 * 64 + 4;

// ---- cache header -------------------------------------------------------------------------------------
struct CacheGeom {
  int L, B, H, D, max_seq, tiles_cap;
  size_t hdr_bytes;      // multiple of 256
  size_t tile_bytes;     // Layout<D>::kTileBytes
  size_t stream_bytes;   // tiles_cap * tile_bytes
  size_t total_bytes;
  size_t off_seq_len, off_arrive, off_status;
  int vq;                   // tq_shape.v_qjl
  size_t vsk_tile_bytes;    // VskLayout<D>::kTileBytes, 0 when off
  size_t vsk_stream_bytes;  // tiles_cap * vsk_tile_bytes
  size_t off_vsk;           // byte offset of the first V-sketch tile
};

inline __host__ bool make_geom(const tq_shape* s, CacheGeom* g) {
  if (!s) return false;
  if (s->n_layers <= 0 || s->batch <= 0 || s->n_heads <= 0 || s->max_seq <= 0) return false;
  if (s->head_dim != 64 && s->head_dim != 128) return false;
  g->L = s->n_layers;
  g->B = s->batch;
  g->H = s->n_heads;
  g->D = s->head_dim;
  g->max_seq = s->max_seq;
  g->tiles_cap = (s->max_seq + kTile - 1) / kTile;
  size_t lb = (size_t)g->L * g->B;
  g->off_seq_len = 0;
  g->off_arrive = lb * 4;
  g->off_status = 2 * lb * 4;
  g->hdr_bytes = ((2 * lb * 4 + 4) + 255) / 256 * 256;
  g->tile_bytes = g->D == 64 ? Layout<64>::kTileBytes : Layout<128>::kTileBytes;
  g->stream_bytes = (size_t)g->tiles_cap * g->tile_bytes;
  g->vq = s->v_qjl == 1;
  g->vsk_tile_bytes = !g->vq ? 0 : (g->D == 64 ? VskLayout<64>::kTileBytes : VskLayout<128>::kTileBytes);
  g->vsk_stream_bytes = (size_t)g->tiles_cap * g->vsk_tile_bytes;
  g->off_vsk = g->hdr_bytes + (size_t)g->L * g->B * g->H * g->stream_bytes;
  g->total_bytes = g->off_vsk + (size_t)g->L * g->B * g->H * g->vsk_stream_bytes;
  return true;
}

// Device-side view passed by value to kernels.
struct CacheView {
  unsigned char* tiles;  // first tile of unit 0
  int32_t* seq_len;      // [L][B]
  int32_t* arrive;       // [L][B]
  int32_t* status;
  int B, H, max_seq, tiles_cap;
  size_t stream_bytes;
  unsigned char* vsk;       // first V-sketch tile of unit 0, or nullptr (v_qjl = 0)
  size_t vsk_stream_bytes;
};

inline __host__ CacheView make_view(const CacheGeom& g, void* data) {
  CacheView v;
  unsigned char* p = (unsigned char*)data;
  v.tiles = p + g.hdr_bytes;
  v.seq_len = (int32_t*)(p + g.off_seq_len);
  v.arrive = (int32_t*)(p + g.off_arrive);
  v.status = (int32_t*)(p + g.off_status);
  v.B = g.B;
  v.H = g.H;
  v.max_seq = g.max_seq;
  v.tiles_cap = g.tiles_cap;
  v.stream_bytes = g.stream_bytes;
  v.vsk = g.vq ? p + g.off_vsk : nullptr;
  v.vsk_stream_bytes = g.vsk_stream_bytes;
  return v;
}


// ---- kernel argument blocks (filled by tq_api.cu, consumed by the launchers) -----------------------------
struct QuantArgs {
  CacheView cv;
  const void* k;  // [B][H][n_tokens][D]  (prefill)  |  [B][H][D] (append)
  const void* v;
  const float* pi_k;  // [H][D][D] of this layer
  const float* pi_v;
  const float* lut_k;  // [H][8] of this layer
  const float* lut_v;
  const float* S;        // [D][D]
  const float* rope_cs;  // [max_seq][D/2][2]
  int layer, n_tokens, start_pos, rope_layout, tiles_per_cta;
  // paper-literal Eq. 6-7 mode (include/tq.h): no normalisation, norm plane 1.0, rnorm plane = e-bar m sqrt(2/pi)
  int literal;
  const float* ebar_k;  // [H] of this layer (literal mode)
};

struct DecodeArgs {
  CacheView cv;
  const float* pi_k;  // [L][H][D][D]
  const float* pi_v;
  const float* lut_k;  // [L][H][8]
  const float* lut_v;
  const float* S;
  const float* rope_cs;
  const void* q;         // [Lc][B][H][D]
  void* out;             // [Lc][B][H][D]
  const int32_t* q_pos;  // [Lc][B] or nullptr
  unsigned* frags;       // workspace [units_call][FragLayout<D>::kWords] (tq_prep.cu)
  unsigned* tabs;        // workspace [layers_call * H][kTabWords]
  float* orot;           // workspace [units_call][D]: o'/l in the rotated basis (tq_decode_model_step)
  float* partials;       // workspace [units_call][64][decode_record_floats(D, v_qjl)]: D + 2 floats, 2 D + 3 with the V sketch
  int* counters;         // workspace [units_call]
  int layer_begin, n_layers_call, nsplit /* CTAs per unit, >= 1 */, per /* tiles per split planned from t_hint */, rope_layout, dt;
  // 0: wait for the kernel in front of this launch before touching memory (any stream order is safe);
  // 1: run ahead — this launch is one of a chain of streaming kernels over DIFFERENT layers whose common producer (the
  //    multi-layer prep kernel) was already awaited by the first of the chain: nothing is awaited at the start, and the
  //    CTAs wait for the kernel in front only before they exit, so that the chain still completes in order.
  int chain_mode;
  int literal;          // paper-literal mode of the append (see QuantArgs)
  const float* ebar_k;  // [L][H]
};

cudaError_t launch_quantize_pack(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st);
cudaError_t launch_quantize_pack_tc(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st);  // tcgen05
cudaError_t launch_prep(const DecodeArgs& d, const void* k, const void* v, int D, int num_sms, bool do_append,
                        bool do_query, cudaStream_t st);
cudaError_t launch_decode(const DecodeArgs& a, int D, bool fused_out, cudaStream_t st);
cudaError_t launch_finish(const DecodeArgs& a, int D, bool programmatic, cudaStream_t st);
int decode_ctas_per_sm(int D);
int decode_record_floats(int D, bool vq);  // floats of one split-K partial record
cudaError_t launch_export(const CacheGeom& g, const CacheView& cv, int layer, int n_tokens, const tq_canonical& out,
                          cudaStream_t st);
cudaError_t launch_import(const CacheGeom& g, const CacheView& cv, int layer, int n_tokens, const tq_canonical& in,
                          cudaStream_t st);

void debug_set_quantize_fp32(int on);

// ---- launch bookkeeping ---------------------------------------------------------------------------------
void count_launch(int n = 1);

// Programmatic dependent launch: the streaming decode kernel is launched with programmatic stream serialization, so
// its CTAs may be scheduled while the prep kernel in front of it is still running; it must call pdl_wait() before it
// reads anything an earlier kernel may have written (only L2 prefetch hints and constants come before that).  The
// prep kernel calls pdl_trigger() to let that happen.  Both are no-ops for ordinary launches.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }

// ---- small device helpers -------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// binary16 bits of x >= 0, round-to-nearest-even, clamped to 65504 (include/tq.h canonical format)
__device__ __forceinline__ unsigned short f32_to_f16_bits_clamped(float x) {
  x = fminf(x, 65504.0f);
  return __half_as_ushort(__float2half_rn(x));
}
__device__ __forceinline__ float f16_bits_to_f32(unsigned short h) { return __half2float(__ushort_as_half(h)); }
// paper-literal mode: the rnorm plane holds e-bar m sqrt(2/pi), rounded to binary16 straight from fp64
__device__ __forceinline__ unsigned short literal_rnorm_bits(float ebar, int m) {
  const double g = fmin((double)ebar * (double)m * 0.79788456080286535588, 65504.0);
  return __half_as_ushort(__double2half(g));
}
constexpr unsigned short kF16One = 0x3C00;

template <typename T>
__device__ __forceinline__ float load_as_float(const T* p);
template <>
__device__ __forceinline__ float load_as_float<float>(const float* p) {
  return *p;
}
template <>
__device__ __forceinline__ float load_as_float<__half>(const __half* p) {
  return __half2float(*p);
}

// y[i] = sum_k M[i][k] x[k] for the rows owned by this warp, all loads of a batch of RB rows issued before
// the first reduction so that the L2 latency is paid once per batch, not once per row.
template <int D, int NWARPS>
__device__ __forceinline__ void matvec_rows_ilp(const float* __restrict__ M, const float* xsm, float* ysm, int warp,
                                                int lane) {
  constexpr int ROWS = D / NWARPS;  // rows per warp
  constexpr int RB = ROWS < 8 ? ROWS : 8;
  constexpr int KP = D / 32;  // elements per lane per row
  float xr[KP];
#pragma unroll
  for (int j = 0; j < KP; ++j) xr[j] = xsm[lane + 32 * j];
#pragma unroll
  for (int r0 = 0; r0 < ROWS; r0 += RB) {
    float m[RB][KP];
#pragma unroll
    for (int r = 0; r < RB; ++r)
#pragma unroll
      for (int j = 0; j < KP; ++j) m[r][j] = __ldg(M + (size_t)(warp * ROWS + r0 + r) * D + lane + 32 * j);
    float p[RB];
#pragma unroll
    for (int r = 0; r < RB; ++r) {
      p[r] = 0.f;
#pragma unroll
      for (int j = 0; j < KP; ++j) p[r] = fmaf(m[r][j], xr[j], p[r]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int r = 0; r < RB; ++r) p[r] += __shfl_xor_sync(0xffffffffu, p[r], o);
    if (lane == 0) {
#pragma unroll
      for (int r = 0; r < RB; ++r) ysm[warp * ROWS + r0 + r] = p[r];
    }
  }
}


}  // namespace tq
