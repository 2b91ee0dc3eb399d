// tq_layout.cu — conversion between the device tile layout and the canonical packed planes
// (include/tq.h "Canonical packed format" / "Device cache format").  Byte shuffling only; not hot.
// Both directions go through the position functions of tq_common.cuh (k_field_pos, sign_bit_pos, v_code_pos).
#include "tq_common.cuh"

namespace tq {

// bits [bit, bit + n) of lane l's word string in a section of W words per lane
__device__ __forceinline__ unsigned sec_get(const unsigned char* sec, int W, int l, int bit, int n) {
  const int w = bit >> 5, s = bit & 31;
  unsigned long long v = *(const unsigned*)(sec + word_offset(W, w, l));
  if (s + n > 32) v |= (unsigned long long)*(const unsigned*)(sec + word_offset(W, w + 1, l)) << 32;
  return (unsigned)((v >> s) & ((1u << n) - 1u));
}
__device__ __forceinline__ void or_bits(unsigned* words, int bit, int n, unsigned val) {
  const int w = bit >> 5, s = bit & 31;
  const unsigned long long v = (unsigned long long)val << s;
  words[w] |= (unsigned)v;
  if (s + n > 32) words[w + 1] |= (unsigned)(v >> 32);
}
// n bits at position `bit` of a canonical LSB-first byte stream
__device__ __forceinline__ unsigned stream_get(const unsigned char* p, int bit, int n) {
  unsigned v = 0;
  for (int k = 0; k < n; ++k) v |= ((p[(bit + k) >> 3] >> ((bit + k) & 7)) & 1u) << k;
  return v;
}

// one thread per (b, h, token): gathers its bits from the lanes that hold them
template <int D>
__global__ void export_kernel(CacheView cv, int layer, int n_tokens, tq_canonical out) {
  using Lo = Layout<D>;
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  const long total = (long)cv.B * cv.H * n_tokens;
  if (idx >= total) return;
  const int t = (int)(idx % n_tokens);
  const long bh = idx / n_tokens;  // b*H + h
  const size_t unit = (size_t)layer * cv.B * cv.H + bh;
  const unsigned char* tile = cv.tiles + unit * cv.stream_bytes + (size_t)(t / kTile) * Lo::kTileBytes;
  const int slot = t % kTile;
  unsigned char* kc = out.k_codes + (size_t)idx * (3 * D / 8);
  unsigned char* vc = out.v_codes + (size_t)idx * (3 * D / 8);
  unsigned char* ks = out.k_signs + (size_t)idx * (D / 8);
  for (int grp = 0; grp < D / 8; ++grp) {  // 8 codes = 4 pair fields = 3 canonical bytes
    unsigned pk = 0, pv = 0;
    for (int q = 0; q < 4; ++q) {
      const BitPos kp = k_field_pos<D>(slot, 4 * grp + q);
      pk |= sec_get(tile + Lo::kOffKC, Lo::KCW, kp.lane, kp.bit, 6) << (6 * q);
    }
    for (int i = 0; i < 8; ++i) {
      const BitPos vp = v_code_pos<D>(slot, 8 * grp + i);
      pv |= sec_get(tile + Lo::kOffVC, Lo::KCW, vp.lane, vp.bit, 3) << (3 * i);
    }
    kc[3 * grp] = pk & 0xff, kc[3 * grp + 1] = (pk >> 8) & 0xff, kc[3 * grp + 2] = (pk >> 16) & 0xff;
    vc[3 * grp] = pv & 0xff, vc[3 * grp + 1] = (pv >> 8) & 0xff, vc[3 * grp + 2] = (pv >> 16) & 0xff;
  }
  for (int byte = 0; byte < D / 8; ++byte) {
    unsigned v = 0;
    for (int k = 0; k < 8; ++k) {
      const BitPos sp = sign_bit_pos<D>(slot, 8 * byte + k);
      v |= sec_get(tile + Lo::kOffKS, Lo::KSW, sp.lane, sp.bit, 1) << k;
    }
    ks[byte] = (unsigned char)v;
  }
  const int nl = slot_lane(slot);
  const unsigned nk = ((const unsigned*)(tile + Lo::kOffNK))[nl];
  out.k_norm[idx] = (unsigned short)(nk & 0xffffu);
  out.k_rnorm[idx] = (unsigned short)(nk >> 16);
  out.v_norm[idx] = ((const unsigned short*)(tile + Lo::kOffVN))[nl];
  if (cv.vsk) {  // V-side sketch tiles
    using Vs = VskLayout<D>;
    const unsigned char* vt = cv.vsk + unit * cv.vsk_stream_bytes + (size_t)(t / kTile) * Vs::kTileBytes;
    unsigned char* vs = out.v_signs + (size_t)idx * (D / 8);
    for (int byte = 0; byte < D / 8; ++byte) {
      unsigned v = 0;
      for (int k = 0; k < 8; ++k) {
        const BitPos sp = vsign_bit_pos<D>(slot, 8 * byte + k);
        v |= sec_get(vt + Vs::kOffVS, Vs::KSW, sp.lane, sp.bit, 1) << k;
      }
      vs[byte] = (unsigned char)v;
    }
    out.v_rnorm[idx] = ((const unsigned short*)(vt + Vs::kOffVR))[nl];
  }
}

// one thread per (b, h, tile, lane): assembles that lane's word strings from the canonical planes; the bits of
// tokens at or beyond n_tokens keep whatever the tile held
template <int D>
__global__ void import_kernel(CacheView cv, int layer, int n_tokens, tq_canonical in) {
  using Lo = Layout<D>;
  const int ntile = (n_tokens + kTile - 1) / kTile;
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  const long total = (long)cv.B * cv.H * ntile * kTile;
  if (idx == 0)
    for (int b = 0; b < cv.B; ++b) cv.seq_len[layer * cv.B + b] = n_tokens;
  if (idx >= total) return;
  const int lane = (int)(idx % kTile), g = lane >> 2, t = lane & 3;
  const int tl = (int)((idx / kTile) % ntile);
  const long bh = idx / ((long)kTile * ntile);
  const size_t unit = (size_t)layer * cv.B * cv.H + bh;
  unsigned char* tile = cv.tiles + unit * cv.stream_bytes + (size_t)tl * Lo::kTileBytes;
  const size_t tok0 = (size_t)bh * n_tokens + (size_t)tl * kTile;  // canonical index of the tile's slot 0
  auto in_call = [&](int s) { return tl * kTile + s < n_tokens; };
  unsigned words[Lo::KCW + 1], keep[Lo::KCW + 1];
  auto flush = [&](unsigned char* sec, int W) {
    for (int w = 0; w < W; ++w) {
      unsigned* p = (unsigned*)(sec + word_offset(W, w, lane));
      *p = (*p & ~keep[w]) | words[w];
    }
  };
  // K codes: slots g + 8 r, pairs t + 4 j
  for (int w = 0; w <= Lo::KCW; ++w) words[w] = 0, keep[w] = 0;
  for (int r = 0; r < 4; ++r) {
    const int s = g + 8 * r;
    if (!in_call(s)) continue;
    const unsigned char* kc = in.k_codes + (tok0 + s) * (3 * D / 8);
    for (int j = 0; j < Lo::J; ++j) {
      const int p = t + 4 * j;
      or_bits(words, k_field_pos<D>(s, p).bit, 6, stream_get(kc, 6 * p, 6));
      or_bits(keep, k_field_pos<D>(s, p).bit, 6, 63u);
    }
  }
  flush(tile + Lo::kOffKC, Lo::KCW);
  // K signs: slots g + 8 r, sketch rows [t d/4, (t + 1) d/4)
  for (int w = 0; w <= Lo::KCW; ++w) words[w] = 0, keep[w] = 0;
  for (int r = 0; r < 4; ++r) {
    const int s = g + 8 * r;
    if (!in_call(s)) continue;
    const unsigned char* ks = in.k_signs + (tok0 + s) * (D / 8);
    for (int i = 0; i < D / 4; ++i) {
      const int rho = t * (D / 4) + i;
      or_bits(words, sign_bit_pos<D>(s, rho).bit, 1, stream_get(ks, rho, 1));
      or_bits(keep, sign_bit_pos<D>(s, rho).bit, 1, 1u);
    }
  }
  flush(tile + Lo::kOffKS, Lo::KSW);
  // V codes: token pairs t + 4 j, coordinates g + 8 c
  for (int w = 0; w <= Lo::KCW; ++w) words[w] = 0, keep[w] = 0;
  for (int j = 0; j < 4; ++j)
    for (int e = 0; e < 2; ++e) {
      const int s = 2 * (t + 4 * j) + e;
      if (!in_call(s)) continue;
      const unsigned char* vc = in.v_codes + (tok0 + s) * (3 * D / 8);
      for (int c = 0; c < Lo::C; ++c) {
        const int i = g + 8 * c;
        or_bits(words, v_code_pos<D>(s, i).bit, 3, stream_get(vc, 3 * i, 3));
        or_bits(keep, v_code_pos<D>(s, i).bit, 3, 7u);
      }
    }
  flush(tile + Lo::kOffVC, Lo::KCW);
  const int s = lane_slot(lane);
  if (in_call(s)) {
    ((unsigned*)(tile + Lo::kOffNK))[lane] = (unsigned)in.k_norm[tok0 + s] | ((unsigned)in.k_rnorm[tok0 + s] << 16);
    ((unsigned short*)(tile + Lo::kOffVN))[lane] = in.v_norm[tok0 + s];
  }
  if (cv.vsk) {  // V-side sketch tiles: this lane's sketch rows g + 8 q of the tokens 2t + e + 8 th + 16 ks
    using Vs = VskLayout<D>;
    unsigned char* vt = cv.vsk + unit * cv.vsk_stream_bytes + (size_t)tl * Vs::kTileBytes;
    for (int w = 0; w <= Lo::KCW; ++w) words[w] = 0, keep[w] = 0;
    for (int sq = 0; sq < 8; ++sq) {
      const int sv = 16 * (sq >> 2) + 8 * ((sq >> 1) & 1) + 2 * t + (sq & 1);
      if (!in_call(sv)) continue;
      const unsigned char* vsg = in.v_signs + (tok0 + sv) * (D / 8);
      for (int q = 0; q < D / 8; ++q) {
        const int rho = g + 8 * q;
        or_bits(words, vsign_bit_pos<D>(sv, rho).bit, 1, stream_get(vsg, rho, 1));
        or_bits(keep, vsign_bit_pos<D>(sv, rho).bit, 1, 1u);
      }
    }
    flush(vt + Vs::kOffVS, Vs::KSW);
    if (in_call(s)) ((unsigned short*)(vt + Vs::kOffVR))[lane] = in.v_rnorm[tok0 + s];
  }
}

cudaError_t launch_export(const CacheGeom& g, const CacheView& cv, int layer, int n_tokens, const tq_canonical& out,
                          cudaStream_t st) {
  long total = (long)g.B * g.H * n_tokens;
  if (total == 0) return cudaSuccess;
  int blocks = (int)((total + 127) / 128);
  if (g.D == 64)
    export_kernel<64><<<blocks, 128, 0, st>>>(cv, layer, n_tokens, out);
  else
    export_kernel<128><<<blocks, 128, 0, st>>>(cv, layer, n_tokens, out);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_import(const CacheGeom& g, const CacheView& cv, int layer, int n_tokens, const tq_canonical& in,
                          cudaStream_t st) {
  long total = (long)g.B * g.H * ((n_tokens + kTile - 1) / kTile) * kTile;
  int blocks = (int)((total + 127) / 128);
  if (blocks == 0) blocks = 1;
  if (g.D == 64)
    import_kernel<64><<<blocks, 128, 0, st>>>(cv, layer, n_tokens, in);
  else
    import_kernel<128><<<blocks, 128, 0, st>>>(cv, layer, n_tokens, in);
  count_launch();
  return cudaGetLastError();
}

}  // namespace tq
