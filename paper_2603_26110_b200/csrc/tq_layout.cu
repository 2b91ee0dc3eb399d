// tq_layout.cu — conversion between the device tile layout and the canonical packed planes
// (include/tq.h "Canonical packed format" / "Device cache format").  Byte shuffling only; not hot.
#include "tq_common.cuh"

namespace tq {

// read/write a 6-bit field at position k of a little-endian word string
__device__ __forceinline__ unsigned get_bits(const unsigned* words, int bitpos, int nbits) {
  int w = bitpos >> 5, s = bitpos & 31;
  unsigned long long v = words[w];
  if (s + nbits > 32) v |= (unsigned long long)words[w + 1] << 32;
  return (unsigned)((v >> s) & ((1u << nbits) - 1u));
}
__device__ __forceinline__ void or_bits(unsigned* words, int bitpos, int nbits, unsigned val) {
  int w = bitpos >> 5, s = bitpos & 31;
  unsigned long long v = (unsigned long long)val << s;
  words[w] |= (unsigned)v;
  if (s + nbits > 32) words[w + 1] |= (unsigned)(v >> 32);
}

template <int D>
__device__ void load_section(const unsigned char* sec, int W, int slot, unsigned* words) {
  for (int w = 0; w < W; ++w) words[w] = *(const unsigned*)(sec + word_offset(W, w, slot));
}
template <int D>
__device__ void store_section(unsigned char* sec, int W, int slot, const unsigned* words) {
  for (int w = 0; w < W; ++w) *(unsigned*)(sec + word_offset(W, w, slot)) = words[w];
}

template <int D>
__global__ void export_kernel(CacheView cv, int layer, int n_tokens, tq_canonical out) {
  using Lo = Layout<D>;
  long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  long total = (long)cv.B * cv.H * n_tokens;
  if (idx >= total) return;
  int t = (int)(idx % n_tokens);
  long bh = idx / n_tokens;  // b*H + h
  size_t unit = (size_t)layer * cv.B * cv.H + bh;
  const unsigned char* tile = cv.tiles + unit * cv.stream_bytes + (size_t)(t / kTile) * Lo::kTileBytes;
  int slot = t % kTile;
  unsigned words[Lo::KCW + 1];
  unsigned char codes[D];
  // K codes: pair group g sits at field position (g - slot) mod P
  load_section<D>(tile + Lo::kOffKC, Lo::KCW, slot, words);
  words[Lo::KCW] = 0;
  for (int g = 0; g < Lo::P; ++g) {
    int k = (g - slot + 4 * Lo::P) % Lo::P;
    unsigned f = get_bits(words, 6 * k, 6);
    codes[2 * g] = f & 7;
    codes[2 * g + 1] = f >> 3;
  }
  unsigned char* kc = out.k_codes + (size_t)idx * (3 * D / 8);
  for (int grp = 0; grp < D / 8; ++grp) {
    unsigned p = 0;
    for (int i = 0; i < 8; ++i) p |= (unsigned)codes[8 * grp + i] << (3 * i);
    kc[3 * grp] = p & 0xff;
    kc[3 * grp + 1] = (p >> 8) & 0xff;
    kc[3 * grp + 2] = (p >> 16) & 0xff;
  }
  // K signs: nibble group n sits at nibble position (n - slot) mod NG
  load_section<D>(tile + Lo::kOffKS, Lo::KSW, slot, words);
  unsigned char* ks = out.k_signs + (size_t)idx * (D / 8);
  for (int byte = 0; byte < D / 8; ++byte) {
    unsigned v = 0;
    for (int half = 0; half < 2; ++half) {
      int n = 2 * byte + half;
      int k = (n - slot + 4 * Lo::NG) % Lo::NG;
      v |= get_bits(words, 4 * k, 4) << (4 * half);
    }
    ks[byte] = (unsigned char)v;
  }
  // V codes: lane g of the tile owns pair groups g (+32 for d = 128); token slot j sits at bits [6j, 6j+6)
  for (int g = 0; g < Lo::P; ++g) {
    const int lane = g % kTile, part = g / kTile;
    const int bit = 192 * part + 6 * slot;
    const unsigned char* sec = tile + Lo::kOffVC;
    unsigned w0 = *(const unsigned*)(sec + word_offset(Lo::KCW, bit >> 5, lane));
    unsigned w1 = ((bit & 31) > 26) ? *(const unsigned*)(sec + word_offset(Lo::KCW, (bit >> 5) + 1, lane)) : 0u;
    unsigned long long v = w0 | ((unsigned long long)w1 << 32);
    unsigned f = (unsigned)(v >> (bit & 31)) & 63u;
    codes[2 * g] = f & 7;
    codes[2 * g + 1] = f >> 3;
  }
  unsigned char* vc = out.v_codes + (size_t)idx * (3 * D / 8);
  for (int grp = 0; grp < D / 8; ++grp) {
    unsigned p = 0;
    for (int i = 0; i < 8; ++i) p |= (unsigned)codes[8 * grp + i] << (3 * i);
    vc[3 * grp] = p & 0xff;
    vc[3 * grp + 1] = (p >> 8) & 0xff;
    vc[3 * grp + 2] = (p >> 16) & 0xff;
  }
  out.k_norm[idx] = ((const unsigned short*)(tile + Lo::kOffKN))[slot];
  out.k_rnorm[idx] = ((const unsigned short*)(tile + Lo::kOffKR))[slot];
  out.v_norm[idx] = ((const unsigned short*)(tile + Lo::kOffVN))[slot];
}

template <int D>
__global__ void import_kernel(CacheView cv, int layer, int n_tokens, tq_canonical in) {
  using Lo = Layout<D>;
  long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  long total = (long)cv.B * cv.H * n_tokens;
  if (idx == 0)
    for (int b = 0; b < cv.B; ++b) cv.seq_len[layer * cv.B + b] = n_tokens;
  if (idx >= total) return;
  int t = (int)(idx % n_tokens);
  long bh = idx / n_tokens;
  size_t unit = (size_t)layer * cv.B * cv.H + bh;
  unsigned char* tile = cv.tiles + unit * cv.stream_bytes + (size_t)(t / kTile) * Lo::kTileBytes;
  int slot = t % kTile;
  unsigned words[Lo::KCW + 1];
  unsigned char codes[D];
  const unsigned char* kc = in.k_codes + (size_t)idx * (3 * D / 8);
  for (int grp = 0; grp < D / 8; ++grp) {
    unsigned p = kc[3 * grp] | ((unsigned)kc[3 * grp + 1] << 8) | ((unsigned)kc[3 * grp + 2] << 16);
    for (int i = 0; i < 8; ++i) codes[8 * grp + i] = (p >> (3 * i)) & 7;
  }
  for (int w = 0; w <= Lo::KCW; ++w) words[w] = 0;
  for (int g = 0; g < Lo::P; ++g) {
    int k = (g - slot + 4 * Lo::P) % Lo::P;
    or_bits(words, 6 * k, 6, codes[2 * g] | ((unsigned)codes[2 * g + 1] << 3));
  }
  store_section<D>(tile + Lo::kOffKC, Lo::KCW, slot, words);
  const unsigned char* ks = in.k_signs + (size_t)idx * (D / 8);
  for (int w = 0; w <= Lo::KSW; ++w) words[w] = 0;
  for (int n = 0; n < Lo::NG; ++n) {
    unsigned nib = (ks[n >> 1] >> (4 * (n & 1))) & 0xf;
    int k = (n - slot + 4 * Lo::NG) % Lo::NG;
    or_bits(words, 4 * k, 4, nib);
  }
  store_section<D>(tile + Lo::kOffKS, Lo::KSW, slot, words);
  // V code words are shared by the 32 tokens of a tile: import_v_kernel (second pass) writes them.
  ((unsigned short*)(tile + Lo::kOffKN))[slot] = in.k_norm[idx];
  ((unsigned short*)(tile + Lo::kOffKR))[slot] = in.k_rnorm[idx];
  ((unsigned short*)(tile + Lo::kOffVN))[slot] = in.v_norm[idx];
}

// V code words of one tile hold all 32 tokens: one thread per (b, h, tile, lane) assembles its words from the
// canonical planes (tokens beyond n_tokens keep whatever the tile held).
template <int D>
__global__ void import_v_kernel(CacheView cv, int layer, int n_tokens, tq_canonical in) {
  using Lo = Layout<D>;
  const int ntile = (n_tokens + kTile - 1) / kTile;
  long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  long total = (long)cv.B * cv.H * ntile * kTile;
  if (idx >= total) return;
  const int lane = (int)(idx % kTile);
  const int tl = (int)((idx / kTile) % ntile);
  const long bh = idx / ((long)kTile * ntile);
  size_t unit = (size_t)layer * cv.B * cv.H + bh;
  unsigned char* sec = cv.tiles + unit * cv.stream_bytes + (size_t)tl * Lo::kTileBytes + Lo::kOffVC;
  unsigned words[Lo::KCW + 1];
  unsigned keep[Lo::KCW + 1];
  for (int w = 0; w <= Lo::KCW; ++w) words[w] = 0, keep[w] = 0;
  for (int part = 0; part < Lo::P / kTile; ++part) {
    const int g = lane + kTile * part;
    for (int j = 0; j < kTile; ++j) {
      const int t = tl * kTile + j;
      if (t >= n_tokens) continue;
      const unsigned char* vc = in.v_codes + ((size_t)bh * n_tokens + t) * (3 * D / 8);
      const int cbit = 6 * g;  // codes 2g, 2g+1 are 6 consecutive bits of the canonical stream
      unsigned v = vc[cbit >> 3] | ((unsigned)vc[(cbit >> 3) + 1 < 3 * D / 8 ? (cbit >> 3) + 1 : (cbit >> 3)] << 8);
      unsigned f = (v >> (cbit & 7)) & 63u;
      or_bits(words, 192 * part + 6 * j, 6, f);
      or_bits(keep, 192 * part + 6 * j, 6, 63u);
    }
  }
  for (int w = 0; w < Lo::KCW; ++w) {
    unsigned* p = (unsigned*)(sec + word_offset(Lo::KCW, w, lane));
    *p = (*p & ~keep[w]) | words[w];
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
  long total = (long)g.B * g.H * n_tokens;
  int blocks = (int)((total + 127) / 128);
  if (blocks == 0) blocks = 1;
  if (g.D == 64)
    import_kernel<64><<<blocks, 128, 0, st>>>(cv, layer, n_tokens, in);
  else
    import_kernel<128><<<blocks, 128, 0, st>>>(cv, layer, n_tokens, in);
  count_launch();
  if (total > 0) {
    long vt = (long)g.B * g.H * ((n_tokens + kTile - 1) / kTile) * kTile;
    int vb = (int)((vt + 127) / 128);
    if (g.D == 64)
      import_v_kernel<64><<<vb, 128, 0, st>>>(cv, layer, n_tokens, in);
    else
      import_v_kernel<128><<<vb, 128, 0, st>>>(cv, layer, n_tokens, in);
    count_launch();
  }
  return cudaGetLastError();
}

}  // namespace tq
