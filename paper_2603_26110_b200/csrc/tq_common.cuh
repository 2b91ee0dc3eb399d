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
// A "section" is a per-token string of W 32-bit words stored chunk-major: 16-byte chunks [c][token], then
// (if W % 4 == 2) one 8-byte chunk [token].
template <int D>
struct Layout {
  static_assert(D == 64 || D == 128, "head_dim must be 64 or 128");
  static constexpr int P = D / 2;            // six-bit pair fields per code string
  static constexpr int NG = D / 4;           // sign nibble groups
  static constexpr int KCW = 3 * D / 32;     // words per K (or V) code string: 6 | 12
  static constexpr int KSW = D / 32;         // words per sign string: 2 | 4
  static constexpr int kCodeBytes = KCW * 4 * kTile;
  static constexpr int kSignBytes = KSW * 4 * kTile;
  static constexpr int kOffKC = 0;
  static constexpr int kOffKS = kOffKC + kCodeBytes;
  static constexpr int kOffVC = kOffKS + kSignBytes;
  static constexpr int kOffKN = kOffVC + kCodeBytes;  // binary16 |k|   [32]
  static constexpr int kOffKR = kOffKN + 2 * kTile;   // binary16 |r_k| [32]
  static constexpr int kOffVN = kOffKR + 2 * kTile;   // binary16 |v|   [32]
  static constexpr int kTileBytes = kOffVN + 2 * kTile;  // 1984 | 3776
  static constexpr int kBytesPerToken = kTileBytes / kTile;
};

// byte offset (inside its section) of word w of the token in slot t, section of W words per token
__host__ __device__ constexpr int word_offset(int W, int w, int t) {
  return (w < (W / 4) * 4) ? ((w / 4) * 16 * kTile + t * 16 + (w % 4) * 4)
                           : ((W / 4) * 16 * kTile + t * 8 + (w - (W / 4) * 4) * 4);
}

// ---- cache header -------------------------------------------------------------------------------------
struct CacheGeom {
  int L, B, H, D, max_seq, tiles_cap;
  size_t hdr_bytes;      // multiple of 256
  size_t tile_bytes;     // Layout<D>::kTileBytes
  size_t stream_bytes;   // tiles_cap * tile_bytes
  size_t total_bytes;
  size_t off_seq_len, off_arrive, off_status;
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
  g->total_bytes = g->hdr_bytes + (size_t)g->L * g->B * g->H * g->stream_bytes;
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
  float* qrot;           // workspace [units_call][2 D]: q'' then z, pre-scaled (tq_prep.cu)
  float* partials;       // workspace [units_call][64][D + 2]
  int* counters;         // workspace [units_call]
  int layer_begin, n_layers_call, nsplit /* CTAs per unit, >= 1 */, per /* tiles per split planned from t_hint */, rope_layout, dt;
  int zero;  // always 0 (see tq_decode.cu: keeps table base registers opaque to ptxas)
};

cudaError_t launch_quantize_pack(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st);
cudaError_t launch_quantize_pack_tc(const QuantArgs& a, int D, tq_dtype dt, int num_sms, cudaStream_t st);  // tcgen05
cudaError_t launch_prep(const DecodeArgs& d, const void* k, const void* v, int D, bool do_append, bool do_query,
                        cudaStream_t st);
cudaError_t launch_decode(const DecodeArgs& a, int D, cudaStream_t st);
int decode_ctas_per_sm(int D);
cudaError_t launch_export(const CacheGeom& g, const CacheView& cv, int layer, int n_tokens, const tq_canonical& out,
                          cudaStream_t st);
cudaError_t launch_import(const CacheGeom& g, const CacheView& cv, int layer, int n_tokens, const tq_canonical& in,
                          cudaStream_t st);

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
