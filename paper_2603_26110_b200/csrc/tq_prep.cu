// tq_prep.cu — the small kernel in front of the streaming decode kernel.
//
// One CTA per (layer-in-call, head, group of BG batch entries) does, depending on the template flags,
//   kAppend : quantize-and-pack ONE new token per batch entry (PAPER.md:111-116 per vector;
//             BASELINE.json:configs[2]): RoPE(k) -> PI_K -> norm, codes, residual -> S r -> bits;
//             PI_V v -> norm, codes; the words are written into the tile slot seq_len[layer][b] and the last head of
//             the batch entry to arrive bumps seq_len;
//   kQuery  : query preparation for the fused decode kernel (Eq. 4 moves PI to the query; north_star):
//             q'' = PI_K RoPE(q), z = S q''  -> workspace, pre-scaled so that logits come out in log2 units.
// tq_append = <true,false>, tq_decode_attn = <false,true>, tq_decode_step = <true,true>.
//
// The work is tiny (five d x d mat-vecs per unit) and the kernel is bound by latency and by re-reading the three
// d x d fp32 matrices of a head: so a CTA keeps them in REGISTERS — three thread groups (PI_K, S, PI_V), TPR = d/64
// threads per matrix row, 64 row elements per thread — fetches them once and applies them to all BG batch entries
// of its head at once (vectors are read from shared memory as broadcast float4).  Four barriers per CTA:
//   inputs + RoPE | PI_K k, PI_K q, PI_V v and their norms | codes, residual, its norm | S r, S q'' | words out.
#include "tq_common.cuh"

namespace tq {

__device__ __forceinline__ int code_of7(float u, const float* lut) {
  int c = 0;
#pragma unroll
  for (int q = 0; q < 7; ++q) c += (u > 0.5f * (lut[q] + lut[q + 1])) ? 1 : 0;
  return c;
}

struct PrepArgs {
  CacheView cv;
  const float *pi_k, *pi_v, *lut_k, *lut_v, *S, *rope_cs;  // full [L][H]... arrays
  const void *q, *k, *v;                                    // [Lc][B][H][D] each (k, v: append; q: query)
  void* out;                                                // [Lc][B][H][D] (zeroed here for empty caches)
  const int32_t* q_pos;                                     // [Lc][B] or nullptr
  unsigned* frags;                                          // workspace [units][FragLayout<D>::kWords]
  unsigned* tabs;                                           // workspace [layers_call * H][kTabWords]
  int layer_begin, rope_layout;
};

template <int D>
struct PrepCfg {
  static constexpr int TPR = D / 64;          // threads per matrix row (64 row elements each)
  static constexpr int GT = D * TPR;          // threads per group: 64 | 256
  static constexpr int BG = D == 64 ? 4 : 2;  // batch entries per CTA
};

// 64 consecutive elements of one matrix row, in registers
struct RowRegs64 {
  float4 m[16];
  __device__ __forceinline__ void load(const float* __restrict__ p) {
#pragma unroll
    for (int c = 0; c < 16; ++c) m[c] = __ldg(reinterpret_cast<const float4*>(p) + c);
  }
  __device__ __forceinline__ void load_shared(const float* p) {  // 16-byte aligned, conflict-free for a 68-float row pitch
#pragma unroll
    for (int c = 0; c < 16; ++c) m[c] = *(reinterpret_cast<const float4*>(p) + c);
  }
  // acc[e] += <row part, x[e] part>, x in shared memory (every lane of a row group reads the same address)
  template <int BG>
  __device__ __forceinline__ void dot(const float* xs /* [BG][stride] */, int stride, float (&acc)[BG]) const {
#pragma unroll
    for (int c = 0; c < 16; ++c) {
#pragma unroll
      for (int e = 0; e < BG; ++e) {
        const float4 x = *reinterpret_cast<const float4*>(xs + e * stride + 4 * c);
        acc[e] = fmaf(m[c].x, x.x, fmaf(m[c].y, x.y, fmaf(m[c].z, x.z, fmaf(m[c].w, x.w, acc[e]))));
      }
    }
  }
};

template <int D, typename T, bool kAppend, bool kQuery>
__global__ void __launch_bounds__((kAppend ? 3 : 2) * PrepCfg<D>::GT) prep_kernel(PrepArgs a, int nbg, int groups_per_cta) {
  using Lo = Layout<D>;
  using Cfg = PrepCfg<D>;
  constexpr int TPR = Cfg::TPR, GT = Cfg::GT, BG = Cfg::BG;
  constexpr int NT = (kAppend ? 3 : 2) * GT;
  constexpr int WG = GT / 32;  // warps per group
  constexpr int HP = D / 2;
  constexpr float kInvSqrtD = D == 64 ? 0.125f : 0.08838834764831845f;
  constexpr float kScaleK = 1.4426950408889634f * kInvSqrtD;             // log2(e) / sqrt(d)
  constexpr float kScaleS = kScaleK * 1.2533141373155003f / (float)D;  // ... * sqrt(pi/2) / m, m = D
  __shared__ __align__(16) float xk[BG][D], xq[BG][D], xv[BG][D], yq[BG][D], rr[BG][D];
  __shared__ unsigned char cK[BG][D], cV[BG][D], bitb[BG][D];
  __shared__ float redk[BG][WG], redv[BG][WG], redr[BG][WG];
  __shared__ float lutK[8], lutV[8];
  __shared__ __align__(16) float zs[BG][D];  // z of the queries (unscaled)
  __shared__ float fscal[BG][4];             // per entry: 2^eq kScaleK, 2^ez kScaleS (fragment scalings)
  __shared__ int s_len0[BG], s_full[BG];

  const int tid = threadIdx.x, lane = tid & 31;
  const int grp = tid / GT, gt = tid % GT, row = gt / TPR, part = gt % TPR, wg = gt >> 5;
  const int B = a.cv.B, H = a.cv.H;
  // one CTA per (layer-in-call, head) and run of groups_per_cta batch groups: the matrix rows are fetched once and
  // stay in registers over the whole run (the multi-layer model step uses long runs, a single layer short ones)
  const int ncta_lh = (nbg + groups_per_cta - 1) / groups_per_cta;
  const int run = (int)blockIdx.x % ncta_lh, lh_c = (int)blockIdx.x / ncta_lh;
  const int lc = lh_c / H, h = lh_c % H;
  const int layer = a.layer_begin + lc;
  const size_t lh = (size_t)layer * H + h;
  const int bg_first = run * groups_per_cta, bg_end = min(nbg, bg_first + groups_per_cta);

  pdl_trigger();  // the streaming kernel behind this one may start its L2 prefetches
  // ---- matrix rows into registers.  d = 64: the CTA copies its (up to) three 16 KB matrices with fully coalesced
  //      16-byte cp.async into shared memory (row pitch 68 floats: a thread-per-row read is then conflict free) and
  //      every thread picks up its row from there; d = 128: straight from global memory (three 64 KB matrices do not fit)
  constexpr bool kStageRows = D == 64;
  constexpr int kPitch = 68;
  extern __shared__ __align__(16) float msm[];  // [groups][D][kPitch] when kStageRows
  RowRegs64 rowreg;
  if (kStageRows) {
    constexpr int NG_ = kAppend ? 3 : 2;
    for (int idx = tid; idx < NG_ * D * (D / 4); idx += NT) {
      const int gsel = idx / (D * (D / 4)), rem = idx % (D * (D / 4)), r = rem / (D / 4), c4 = rem % (D / 4);
      const float* M = gsel == 0 ? a.pi_k + lh * D * D : gsel == 1 ? a.S : a.pi_v + lh * D * D;
      const unsigned dst = (unsigned)__cvta_generic_to_shared(msm + ((size_t)gsel * D + r) * kPitch + 4 * c4);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(M + (size_t)r * D + 4 * c4) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  } else {
    const float* M = grp == 0 ? a.pi_k + lh * D * D : grp == 1 ? a.S : a.pi_v + lh * D * D;
    rowreg.load(M + (size_t)row * D + part * 64);
  }
  if (tid < 8) lutK[tid] = a.lut_k[lh * 8 + tid];
  if (tid >= 32 && tid < 40) lutV[tid - 32] = a.lut_v[lh * 8 + tid - 32];
  for (int bgi = bg_first; bgi < bg_end; ++bgi) {
  const int b0 = bgi * BG, nb = min(BG, B - b0);
  // ---- the cache lengths first: the RoPE positions and the target tile slot hang off them
  int len_e[BG];
#pragma unroll
  for (int e = 0; e < BG; ++e) len_e[e] = e < nb ? __ldcg(a.cv.seq_len + layer * B + b0 + e) : 0;
  // ---- stage-4 work item of this thread (one 16-bit or 8-bit piece of one token in the device tile layout,
  //      tq_common.cuh), and an early read of the V halfword it will modify (a V field is shared with the other token
  //      of the pair, which was appended by an earlier call)
  constexpr int HW = 3 * D / 64;  // halfwords per (lane, token) block of K fields, and per (lane, token pair) block of V fields
  constexpr int IT_K = 4 * HW, IT_S = 4 * Lo::U * 2, IT_V = 8 * HW;
  constexpr int ITEMS = IT_K + IT_S + IT_V + 1;
  static_assert(!kAppend || BG * ITEMS <= NT, "one output item per thread");
  const int it_e = tid / ITEMS, it = tid % ITEMS;
  int it_len = len_e[0];
#pragma unroll
  for (int j = 1; j < BG; ++j) it_len = it_e == j ? len_e[j] : it_len;
  const bool it_on = kAppend && it_e < nb && it_len < a.cv.max_seq;
  unsigned char* it_tp = a.cv.tiles + (((size_t)layer * B + b0 + min(it_e, nb - 1)) * H + h) * a.cv.stream_bytes +
                         (size_t)(min(it_len, a.cv.max_seq - 1) / kTile) * Lo::kTileBytes;
  const int it_slot = it_len % kTile;
  unsigned short vold = 0;
  unsigned short* vptr = nullptr;
  if (it_on && it >= IT_K + IT_S && it < IT_K + IT_S + IT_V) {
    const int vi = it - IT_K - IT_S, gi = vi / HW, hw = vi % HW, pp = it_slot >> 1;
    const int hidx = (pp >> 2) * HW + hw;  // halfword of lane (gi, pp & 3)'s V string
    vptr = reinterpret_cast<unsigned short*>(it_tp + Lo::kOffVC + word_offset(Lo::KCW, hidx >> 1, 4 * gi + (pp & 3))) + (hidx & 1);
    vold = __ldcg(vptr);
  }

  // ---- inputs of the BG batch entries of this head, RoPE applied to k and q (positions read on the device)
  for (int idx = tid; idx < BG * HP; idx += NT) {
    const int e = idx / HP, g = idx % HP;
    const int ia = a.rope_layout == 0 ? 2 * g : g, ib = a.rope_layout == 0 ? 2 * g + 1 : g + HP;
    float ka = 0.f, kb = 0.f, qa = 0.f, qb = 0.f;
    if (e < nb) {
      const int b = b0 + e;
      int len0 = len_e[0];
#pragma unroll
      for (int j = 1; j < BG; ++j) len0 = e == j ? len_e[j] : len0;
      const bool full = kAppend && len0 >= a.cv.max_seq;
      const int len1 = (kAppend && !full) ? len0 + 1 : len0;  // length the decode kernel will see
      const size_t uc = ((size_t)lc * B + b) * H + h;
      if (g == 0) {
        s_len0[e] = len0;
        s_full[e] = full;
      }
      if (kAppend) {  // the appended key sits at index len0
        const int kpos = min(len0, a.cv.max_seq - 1);
        const T* kp = reinterpret_cast<const T*>(a.k) + uc * D;
        const float xa = load_as_float<T>(kp + ia), xb = load_as_float<T>(kp + ib);
        const float2 cs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)kpos * HP + g) * 2);
        ka = xa * cs.x - xb * cs.y;
        kb = xa * cs.y + xb * cs.x;
      }
      if (kQuery) {  // the query defaults to the newest cached token
        int qpos = a.q_pos ? a.q_pos[lc * B + b] : len1 - 1;
        qpos = max(0, min(qpos, a.cv.max_seq - 1));
        const T* qp = reinterpret_cast<const T*>(a.q) + uc * D;
        const float xa = load_as_float<T>(qp + ia), xb = load_as_float<T>(qp + ib);
        const float2 cs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)qpos * HP + g) * 2);
        qa = xa * cs.x - xb * cs.y;
        qb = xa * cs.y + xb * cs.x;
        if (len1 <= 0) {  // empty cache: no tile for this unit in the streaming kernel, out = 0
          T* outp = reinterpret_cast<T*>(a.out) + uc * D;
          if constexpr (sizeof(T) == 2) outp[ia] = outp[ib] = __float2half_rn(0.f);
          else outp[ia] = outp[ib] = 0.f;
        }
      }
    }
    if (kAppend) xk[e][ia] = ka, xk[e][ib] = kb;
    if (kQuery) xq[e][ia] = qa, xq[e][ib] = qb;
  }
  if (kAppend) {
    for (int idx = tid; idx < BG * D; idx += NT) {
      const int e = idx / D, i = idx % D;
      xv[e][i] = e < nb ? load_as_float<T>(reinterpret_cast<const T*>(a.v) + (((size_t)lc * B + b0 + e) * H + h) * D + i) : 0.f;
    }
  }
  if (kStageRows && bgi == bg_first) asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  if (kStageRows && bgi == bg_first) rowreg.load_shared(msm + ((size_t)grp * D + row) * kPitch);

  // ---- stage 1: rotations (groups 0 and 2) and the norms of the rotated key / value
  float yk[BG], yv[BG];
  if (grp == 0) {
    float aq[BG];
#pragma unroll
    for (int e = 0; e < BG; ++e) yk[e] = 0.f, aq[e] = 0.f;
    if (kAppend) rowreg.dot<BG>(&xk[0][part * 64], D, yk);
    if (kQuery) rowreg.dot<BG>(&xq[0][part * 64], D, aq);
#pragma unroll
    for (int e = 0; e < BG; ++e) {
      if (TPR == 2) {
        yk[e] += __shfl_xor_sync(0xffffffffu, yk[e], 1);
        aq[e] += __shfl_xor_sync(0xffffffffu, aq[e], 1);
      }
      if (kAppend) {
        const float ss = warp_sum(part == 0 ? yk[e] * yk[e] : 0.f);
        if (lane == 0) redk[e][wg] = ss;
      }
      if (kQuery && part == 0) {
        yq[e][row] = aq[e];
      }
    }
  } else if (kAppend && grp == 2) {
#pragma unroll
    for (int e = 0; e < BG; ++e) yv[e] = 0.f;
    rowreg.dot<BG>(&xv[0][part * 64], D, yv);
#pragma unroll
    for (int e = 0; e < BG; ++e) {
      if (TPR == 2) yv[e] += __shfl_xor_sync(0xffffffffu, yv[e], 1);
      const float ss = warp_sum(part == 0 ? yv[e] * yv[e] : 0.f);
      if (lane == 0) redv[e][wg] = ss;
    }
  }
  __syncthreads();

  // ---- stage 2 (append): unit vectors, codes, residual and its norm
  if (kAppend) {
    if (grp == 0 && part == 0) {
#pragma unroll
      for (int e = 0; e < BG; ++e) {
        float n2 = 0.f;
#pragma unroll
        for (int w = 0; w < WG; ++w) n2 += redk[e][w];
        const float n = sqrtf(n2);
        const float u = n > 0.f ? yk[e] / n : 0.f;
        const int c = code_of7(u, lutK);
        const float r = u - lutK[c];
        cK[e][row] = (unsigned char)c;
        rr[e][row] = r;
        yk[e] = r * r;
      }
    }
    if (grp == 0) {  // whole warps: the shuffles need every lane
#pragma unroll
      for (int e = 0; e < BG; ++e) {
        const float ss = warp_sum(part == 0 ? yk[e] : 0.f);
        if (lane == 0) redr[e][wg] = ss;
      }
    } else if (grp == 2 && part == 0) {
#pragma unroll
      for (int e = 0; e < BG; ++e) {
        float n2 = 0.f;
#pragma unroll
        for (int w = 0; w < WG; ++w) n2 += redv[e][w];
        const float n = sqrtf(n2);
        const float u = n > 0.f ? yv[e] / n : 0.f;
        cV[e][row] = (unsigned char)code_of7(u, lutV);
      }
    }
    __syncthreads();
  }

  // ---- stage 3: sketch of the residual (bits) and of the rotated query (z)
  if (grp == 1) {
    float sr[BG], zq[BG];
#pragma unroll
    for (int e = 0; e < BG; ++e) sr[e] = 0.f, zq[e] = 0.f;
    if (kAppend) rowreg.dot<BG>(&rr[0][part * 64], D, sr);
    if (kQuery) rowreg.dot<BG>(&yq[0][part * 64], D, zq);
#pragma unroll
    for (int e = 0; e < BG; ++e) {
      if (TPR == 2) {
        sr[e] += __shfl_xor_sync(0xffffffffu, sr[e], 1);
        zq[e] += __shfl_xor_sync(0xffffffffu, zq[e], 1);
      }
      if (part == 0) {
        if (kAppend) bitb[e][row] = sr[e] >= 0.f ? 1 : 0;
        if (kQuery) zs[e][row] = zq[e];
      }
    }
  }
  __syncthreads();
  if (kQuery) {
    // ---- the decode kernel's operands (tq_common.cuh FragLayout): power-of-two scalings that put max |q''_s|, max |z_s|
    //      in [2^13, 2^14), fp16 hi + lo splits in B-fragment order; and the head's dequantisation tables
    using FL = FragLayout<D>;
    const int warp_id = tid >> 5;
    if (warp_id < BG) {  // one warp per entry: maxima and the sum of z
      const int e = warp_id;
      float qm = 0.f, zm = 0.f, zsum = 0.f;
#pragma unroll
      for (int i = lane; i < D; i += 32) {
        qm = fmaxf(qm, fabsf(yq[e][i] * kScaleK));
        const float zv = zs[e][i] * kScaleS;
        zm = fmaxf(zm, fabsf(zv));
        zsum += zv;
      }
      qm = warp_max(qm), zm = warp_max(zm), zsum = warp_sum(zsum);
      auto expo = [](float x) {
        const int E = (int)((__float_as_uint(x) >> 23) & 0xffu);
        return (E == 0 || E == 255) ? 0 : E - 127;
      };
      auto p2 = [](int ee) { return __uint_as_float((unsigned)(max(-100, min(100, ee)) + 127) << 23); };
      const int eq = 13 - expo(qm), ez = 13 - expo(zm);
      if (lane == 0) {
        fscal[e][0] = p2(eq) * kScaleK;
        fscal[e][1] = p2(ez) * kScaleS;
        if (e < nb) {
          float* sc = reinterpret_cast<float*>(a.frags + (((size_t)lc * B + b0 + e) * H + h) * FL::kWords + FL::kScalOff);
          sc[0] = p2(-eq), sc[1] = p2(25 - ez), sc[2] = zsum, sc[3] = 0.f;
        }
      }
    }
    __syncthreads();
    auto split2 = [](float x0, float x1, bool lo) {
      const __half h0 = __float2half_rn(x0), h1 = __float2half_rn(x1);
      const __half l0 = __float2half_rn(x0 - __half2float(h0)), l1 = __float2half_rn(x1 - __half2float(h1));
      return lo ? ((unsigned)__half_as_ushort(l0) | ((unsigned)__half_as_ushort(l1) << 16))
                : ((unsigned)__half_as_ushort(h0) | ((unsigned)__half_as_ushort(h1) << 16));
    };
    for (int idx = tid; idx < BG * FL::kScalOff; idx += NT) {
      const int e = idx / FL::kScalOff, wi = idx % FL::kScalOff;
      if (e >= nb) continue;
      const int pat = wi / FL::kWordsPerPat, wd = wi % FL::kWordsPerPat, t = pat & 3;
      const bool lo = pat >> 2;
      unsigned word;
      if (wd < 2 * FL::KS) {
        const int c0 = 16 * (wd >> 1) + 2 * t + 8 * (wd & 1);
        word = split2(yq[e][c0] * fscal[e][0], yq[e][c0 + 1] * fscal[e][0], lo);
      } else {
        const int ks = (wd - 2 * FL::KS) >> 1, reg = wd & 1, p0 = 2 * (ks & 3);
        const int rho = t * (D / 4) + 16 * (ks >> 2) + p0 + reg;
        const float sc = fscal[e][1] * __uint_as_float((unsigned)(127 - p0 - reg) << 23);
        word = split2(zs[e][rho] * sc, zs[e][rho + 8] * sc, lo);
      }
      a.frags[(((size_t)lc * B + b0 + e) * H + h) * FL::kWords + wi] = word;
    }
    if (tid < 64 && bgi == bg_first) {  // every CTA of the head writes the same values
      const int c0 = tid & 7, c1 = tid >> 3;
      unsigned* tb = a.tabs + (size_t)lh_c * kTabWords;
      tb[tid] = split2(lutK[c0], lutK[c1], false);
      tb[64 + tid] = split2(lutK[c0], lutK[c1], true);
      tb[128 + tid] = split2(lutV[c0], lutV[c1], false);
      tb[192 + tid] = split2(lutV[c0], lutV[c1], true);
      if (tid == 0) {
        bool exact = true;
#pragma unroll
        for (int i = 0; i < 8; ++i)
          exact = exact && __half2float(__float2half_rn(lutK[i])) == lutK[i] && __half2float(__float2half_rn(lutV[i])) == lutV[i];
        tb[256] = exact ? 1u : 0u;
      }
    }
  }
  if (!kAppend) {
    __syncthreads();  // the next group of the run reuses the shared arrays
    continue;
  }

  // ---- stage 4 (append): every thread assembles one piece of one token in the device tile layout
  if (it_on) {
    const int e = it_e, slot = it_slot, g = slot & 7, r = slot >> 3;
    unsigned char* tp = it_tp;
    // bits [16 hw, 16 hw + 16) of a string of NB-bit pieces at stride 6 bits: piece k = val(k) at bit 6 k + off
    auto gather16 = [&](int hw, int nfields, int off, int nb_, auto val, unsigned& out, unsigned& mask) {
      out = 0, mask = 0;
      for (int k = 0; k < nfields; ++k) {
        const int sh = 6 * k + off - 16 * hw;
        if (sh <= -nb_ || sh >= 16) continue;
        const unsigned v = val(k), mk = (1u << nb_) - 1u;
        out |= sh >= 0 ? (v << sh) : (v >> (-sh));
        mask |= sh >= 0 ? (mk << sh) : (mk >> (-sh));
      }
      out &= 0xffffu, mask &= 0xffffu;
    };
    if (it < IT_K) {  // K pair fields of lane (g, t): pairs t + 4 j, block r of the lane's string
      const int t = it / HW, hw = it % HW;
      unsigned v, mk;
      gather16(hw, Lo::J, 0, 6, [&](int j) { const int p = t + 4 * j; return (unsigned)(cK[e][2 * p] | (cK[e][2 * p + 1] << 3)); }, v, mk);
      const int hidx = r * HW + hw;
      reinterpret_cast<unsigned short*>(tp + Lo::kOffKC + word_offset(Lo::KCW, hidx >> 1, 4 * g + t))[hidx & 1] = (unsigned short)v;
    } else if (it < IT_K + IT_S) {  // sign bytes: lane (g, t), piece u, byte half hb
      const int si = it - IT_K, t = si / (2 * Lo::U), u = (si / 2) % Lo::U, hb = si & 1;
      unsigned v = 0;
      for (int k = 0; k < 8; ++k) v |= (unsigned)bitb[e][t * (D / 4) + 16 * u + 8 * hb + k] << k;
      const int word = (slot >> 4) * Lo::U + u, byte = 2 * hb + (r & 1);
      *(tp + Lo::kOffKS + word_offset(Lo::KSW, word, 4 * g + t) + byte) = (unsigned char)v;
    } else if (it < IT_K + IT_S + IT_V) {  // V codes: lane (gi, pp & 3), three-bit slices at 6 c + 3 (slot & 1)
      const int vi = it - IT_K - IT_S, gi = vi / HW, hw = vi % HW;
      unsigned v, mk;
      gather16(hw, Lo::C, 3 * (slot & 1), 3, [&](int c) { return (unsigned)cV[e][gi + 8 * c]; }, v, mk);
      *vptr = (unsigned short)((vold & ~mk) | v);
    } else {
      float nk = 0.f, nr = 0.f, nv = 0.f;
#pragma unroll
      for (int w = 0; w < WG; ++w) nk += redk[e][w], nr += redr[e][w], nv += redv[e][w];
      const int nl = slot_lane(slot);
      reinterpret_cast<unsigned*>(tp + Lo::kOffNK)[nl] =
          (unsigned)f32_to_f16_bits_clamped(sqrtf(nk)) | ((unsigned)f32_to_f16_bits_clamped(sqrtf(nr)) << 16);
      reinterpret_cast<unsigned short*>(tp + Lo::kOffVN)[nl] = f32_to_f16_bits_clamped(sqrtf(nv));
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
  __syncthreads();  // the next group of the run reuses the shared arrays
  }  // batch groups of this CTA's run
}

template <int D, typename T>
static cudaError_t launch_prep_t(const PrepArgs& a, int lh_count, int B, int num_sms, bool do_append, bool do_query,
                                 cudaStream_t st) {
  using Cfg = PrepCfg<D>;
  const int nbg = (B + Cfg::BG - 1) / Cfg::BG;
  // batch groups per CTA: a CTA re-uses its matrix rows over a run of groups.  Enough CTAs to fill the GPU twice
  // (a single layer: one group per CTA, shortest latency); the rest of the batch goes into longer runs.
  int gpc = (int)(((long)lh_count * nbg + 2L * num_sms - 1) / (2L * num_sms));
  gpc = gpc < 1 ? 1 : (gpc > nbg ? nbg : gpc);
  const int grid = lh_count * ((nbg + gpc - 1) / gpc);
  const size_t sm3 = D == 64 ? (size_t)3 * D * 68 * 4 : 0, sm2 = D == 64 ? (size_t)2 * D * 68 * 4 : 0;
  if (D == 64) {  // per launch: the attribute is per device and a process may drive several
    cudaError_t e1 = cudaFuncSetAttribute(prep_kernel<D, T, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm3);
    cudaError_t e2 = cudaFuncSetAttribute(prep_kernel<D, T, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm3);
    if (e1 != cudaSuccess) return e1;
    if (e2 != cudaSuccess) return e2;
  }
  if (do_append && do_query) prep_kernel<D, T, true, true><<<grid, 3 * Cfg::GT, sm3, st>>>(a, nbg, gpc);
  else if (do_append) prep_kernel<D, T, true, false><<<grid, 3 * Cfg::GT, sm3, st>>>(a, nbg, gpc);
  else prep_kernel<D, T, false, true><<<grid, 2 * Cfg::GT, sm2, st>>>(a, nbg, gpc);
  count_launch();
  return cudaGetLastError();
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
  const int lh_count = d.n_layers_call * d.cv.H;
  if (D == 64)
    return d.dt == TQ_F16 ? launch_prep_t<64, __half>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st)
                          : launch_prep_t<64, float>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st);
  return d.dt == TQ_F16 ? launch_prep_t<128, __half>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st)
                        : launch_prep_t<128, float>(a, lh_count, d.cv.B, num_sms, do_append, do_query, st);
}

}  // namespace tq
