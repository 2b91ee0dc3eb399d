/*
 * tq.h — C ABI of the B200-native TurboESM hot path (arxiv/paper_2603_26110).
 *
 * Two operations, defined by the paper and by BASELINE.json:north_star:
 *
 *  (a) KV quantize-and-pack  [PAPER.md:111-116 prefill pipeline steps 1,3,4; §3.3 Eq. 5; §3.4 Eq. 6;
 *      §4.2 packing snippet PAPER.md:203-213]: per vector, RoPE (keys only, Eq. 1-2) -> rotate by the
 *      per-(layer, head) orthogonal PI (Eq. 4) -> store the norm -> code every coordinate of the unit
 *      vector against an 8-point Lloyd-Max LUT (separate K and V tables) -> pack at
 *      3 bits per coordinate -> residual r = u - lut[code], store sign(S r) (1 bit per row of S) and |r|.
 *  (b) fused decode attention  [PAPER.md:118-124 decode pipeline, Algorithm 1 PAPER.md:223-237]: rotate
 *      the query once (q'' = PI_K RoPE(q), z = S q''), stream the packed cache, per cached token
 *      logit = n * ( <q'', lut_K[codes]> + sqrt(pi/2)/m * |r| * <z, sigma> ) / sqrt(d), online softmax,
 *      accumulate p * n_v * lut_V[codes_v]; out = PI_V^T (o / l).  No fp16 K or V tensor is ever formed.
 *
 * Conventions
 *  - Every call returns a tq_status.  Argument validation is synchronous on the host; kernels are
 *    launched asynchronously on the given CUDA stream; nothing here calls cudaDeviceSynchronize and
 *    nothing here allocates or frees device memory: the caller owns every buffer.
 *  - "HOST" / "DEVICE" beside a pointer says where it must live.  Device pointers must be 16-byte aligned.
 *  - There is no CPU fallback: with no usable CUDA device every device entry point returns TQ_ERR_CUDA.
 *  - Matrices are row-major.  y = PI x means y[i] = sum_k PI[i*d + k] * x[k].
 *
 * Canonical packed format (what the paper fixes; the oracle emits exactly this; PAPER.md:203-213,
 * tightened to 3 bit/coordinate per BASELINE.json:north_star):
 *   codes : per vector 3d/8 bytes; bit (3i + b) of the LSB-first bit stream = bit b of code_i
 *           (each 8-code group = 3 bytes = the low 24 bits of the paper's INT32 container);
 *   signs : per key vector m/8 bytes; bit j of the LSB-first stream = [ (S r)_j >= 0 ];
 *   norm  : IEEE binary16 bits of |PI x'| (round-to-nearest-even, clamped to 65504);
 *   rnorm : IEEE binary16 bits of |r| (keys only), r taken on the unit vector.
 *
 * Device cache format (opaque to callers; tq_cache_export_canonical / tq_cache_import_canonical convert):
 *   tokens are grouped in tiles of TQ_TILE_TOKENS = 32 and every (layer, batch, head) owns one contiguous
 *   stream of ceil(max_seq/32) tiles.  The fused decode kernel runs its contractions as warp-level tensor-core MMAs
 *   (mma.sync.m16n8k16), so a tile stores every word in the order of the MMA A-fragment: "lane" = 4 g + t, g = lane / 4
 *   the fragment row, t = lane % 4 the fragment column group; per-lane word strings are stored chunk-major
 *   ([16-byte chunk][lane]) so that lane-wise 128-bit reads are contiguous:
 *     K codes : lane (g, t) holds, for the token slots g, g + 8, g + 16, g + 24, the six-bit fields
 *               (code_{2p} | code_{2p+1} << 3) of the coordinate pairs p = t, t + 4, t + 8, ...;
 *     K signs : lane (g, t) holds sketch rows [t m/4, (t+1) m/4) of the same four slots in 16-bit pieces; the pieces of
 *               slots s and s + 8 are byte-interleaved in one 32-bit word so that (word >> 8 ab) & (0x00010001 << p) is an
 *               fp16 pair whose halves are 0 or the subnormal 2^(p-24): the sign bits feed the MMA without unpacking;
 *     V codes : lane (g, t) holds coordinates g, g + 8, g + 16, ... of the token pairs t, t + 4, t + 8, t + 12 as six-bit
 *               fields code(token 2pp) | code(token 2pp + 1) << 3;
 *     norms   : one u32 per lane (binary16 |k| | binary16 |r_k| << 16) and one u16 (binary16 |v|); lane (g, t) owns
 *               slot g + 8 t.
 *   Bytes per cached token-head: 62 (d = 64), 118 (d = 128) — the same as the canonical format.
 *   With v_qjl = 1 every (layer, batch, head) owns a second stream of 32-token tiles for the value sketch (sign bits in
 *   the A-fragment order of the sketch accumulation, binary16 |r_v|): + 10 / 18 bytes per token-head.
 *   A cache has ONE writer at a time: tq_quantize_pack / tq_append / tq_decode_step / tq_decode_model_step /
 *   tq_cache_import_canonical calls that touch the same layer must be ordered by the caller (same stream, or events);
 *   concurrent readers (tq_decode_attn, export) of a layer that is not being written are fine.
 */
#ifndef TQ_H_
#define TQ_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TQ_TILE_TOKENS 32

typedef enum {
  TQ_OK = 0,
  TQ_ERR_INVALID_ARG = 1, /* NULL / misaligned pointer, negative size, layer out of range, ...          */
  TQ_ERR_UNSUPPORTED = 2, /* head_dim not in {64,128}, qjl_dim != head_dim, v_qjl = 1 with residual_mode = 1 */
  TQ_ERR_CAPACITY = 3,    /* host-visible: start_pos + n_tokens > max_seq; workspace / buffer too small   */
  TQ_ERR_CUDA = 4         /* a CUDA runtime call or launch failed (or no device)                         */
} tq_status;

typedef enum { TQ_F16 = 0, TQ_F32 = 1 } tq_dtype;

/* Plain data, caller-filled, passed by pointer, never retained. */
typedef struct {
  int32_t n_layers;    /* L                                                                             */
  int32_t batch;       /* B                                                                             */
  int32_t n_heads;     /* H                                                                             */
  int32_t head_dim;    /* d: 64 or 128                                                                  */
  int32_t qjl_dim;     /* m: must equal head_dim                                                        */
  int32_t max_seq;     /* cache capacity in tokens per (layer, batch, head)                             */
  float rope_base;     /* theta_g = rope_base^(-2g/d); 10000 in BASELINE.json:configs[0]                */
  int32_t rope_layout; /* 0 = interleaved pairs (2g, 2g+1) [PAPER.md:102, Eq. 2]; 1 = half-split (g, g+d/2) */
  int32_t v_qjl;       /* 0 = K-only residual sketch (reading D3); 1 = values carry one too [Algorithm 1
                          line 10, PAPER.md:234]: bits sign(S r_v) and binary16 |r_v| per token, +m/8 + 2 bytes; a
                          dequantised value is then n_v (lut_V[codes] + sqrt(pi/2)/m |r_v| S^T sigma_v).  Not combined
                          with residual_mode 1 (TQ_ERR_UNSUPPORTED)                                              */
  int32_t residual_mode; /* 0 = north_star form: unit vector coded, |y| and |r| stored per token, bits = sign(S r);
                            1 = the paper's literal Eq. 6-7 [PAPER.md:170-179]: see "Paper-literal mode" below   */
} tq_shape;

/* Calibration arrays.  HOST pointers for tq_calibrate_host, DEVICE pointers for every other call.     */
typedef struct {
  float *pi_k;    /* [L][H][d][d]  PI_K, orthogonal, y = PI x                                           */
  float *pi_v;    /* [L][H][d][d]  PI_V                                                                 */
  float *lut_k;   /* [L][H][8]     ascending Lloyd-Max centroids for unit-norm rotated keys             */
  float *lut_v;   /* [L][H][8]     same for values                                                      */
  float *S;       /* [m][d]        QJL sketch matrix, shared by all layers and heads                    */
  float *rope_cs; /* [max_seq][d/2][2]  (cos, sin)(p * theta_g), evaluated in fp64 and rounded to fp32  */
  float *ebar_k;  /* [L][H]  residual_mode 1 only (else may be NULL): the pre-calibrated mean absolute residual of the
                     keys of that head, the scalar of Eq. 7 [PAPER.md:176-179]                                     */
} tq_params;

/* Paper-literal mode (tq_shape.residual_mode = 1).  The paper's own residual correction
 * [PAPER.md:170-179, Eq. 6-7] stores s = sign(x - x^) per coordinate and reconstructs x~ = x^ + s e-bar with one
 * pre-calibrated scalar e-bar per head; its LUTs are calibrated on the raw rotated activations (no norm is stored) and
 * values are not rotated [PAPER.md:157-162].  In this mode tq_quantize_pack / tq_append
 *   - do NOT normalise: codes are taken on y = PI x' itself (LUT entries live on the scale of the activations), and the
 *     stored binary16 norm is exactly 1.0 for keys and values;
 *   - take the residual e = y - lut[code] and store bits_j = [(S e)_j >= 0];
 *   - store, in place of |r|, the binary16 rounding (from fp64) of  e-bar[layer][head] * m * sqrt(2/pi),
 * so that the decode kernel's correction term  sqrt(pi/2)/m * (stored) * <S q'', sigma>  equals  e-bar <S q'', sigma>.
 * With S = I and PI_V = I passed as data (what tq_calibrate_host emits in this mode) this is Eq. 6-7 word for word:
 * bits = sign(e), logit = <q'', lut[codes] + s e-bar> / sqrt(d).  tq_decode_attn itself is the same in both modes.   */

/* Packed cache: one caller-allocated DEVICE buffer of tq_cache_bytes() bytes, zero-filled by the caller
 * before first use.  It holds a header (seq_len[L][B], append arrival counters, a sticky status word)
 * followed by the token tiles.                                                                        */
typedef struct {
  void *data; /* DEVICE, 256-byte aligned */
} tq_cache;

/* ---- sizes (pure host arithmetic; return 0 on an invalid shape) ---------------------------------- */
size_t tq_cache_bytes(const tq_shape *shape);
size_t tq_cache_bytes_per_token_head(const tq_shape *shape); /* 62 or 118; 72 or 136 with v_qjl = 1        */
/* Byte offset inside tq_cache.data of int32 seq_len[L][B] (tokens currently cached) and of the
 * int32 sticky status word (0, or TQ_ERR_CAPACITY once an append was refused on the device).          */
size_t tq_cache_seq_len_offset(const tq_shape *shape);
size_t tq_cache_status_offset(const tq_shape *shape);
/* Workspace for tq_decode_attn / tq_decode_step (n_layers_call = the call's) and tq_decode_model_step (its
 * n_layers_call): the decode kernel's query operands and dequantisation tables, split-K partials, arrival
 * counters.  Must be zero-filled once by the caller; every call leaves it reusable.  Calls that share a
 * workspace must be ordered on one stream.                                                               */
size_t tq_decode_workspace_bytes(const tq_shape *shape, int32_t n_layers_call);
/* Canonical plane sizes in bytes for n_tokens tokens of every (layer?, batch, head) of ONE layer:
 * plane 0 k_codes, 1 k_signs, 2 k_norm, 3 k_rnorm, 4 v_codes, 5 v_norm, 6 v_signs, 7 v_rnorm (6, 7: v_qjl = 1). */
size_t tq_canonical_plane_bytes(const tq_shape *shape, int32_t plane, int32_t n_tokens);

/* ---- host-side calibration (not hot) [PAPER.md:128-143 §3.2; 145-164 §3.3; north_star] ------------
 * Fills out_host (all HOST arrays, caller-allocated with the sizes given in tq_params).
 *  mode 0: PI = V^T from the SVD of the uncentred sample matrix X (n_samples x d) per (layer, head)
 *          [PAPER.md:132-137]; LUTs by Lloyd-Max (1-D k-means) on the pooled coordinates of the
 *          normalised rotated samples.
 *  mode 1: PI = Q of the QR factorisation of a seeded Gaussian d x d matrix (columns sign-fixed so that
 *          diag(R) > 0) [BASELINE.json:configs[0]]; LUTs = Lloyd-Max fixed point for N(0, 1/d) [configs[0]].
 *          k_samples / v_samples may be NULL.
 * S: seeded i.i.d. N(0,1).  rope_cs: fp64 evaluation rounded to fp32.
 * residual_mode 1 (paper-literal): S = I, PI_V = I; the LUTs are fitted to the raw rotated coordinates (mode 0) or stay
 * the N(0, 1/d) tables (mode 1); ebar_k (required) = the mean absolute residual of the keys under lut_k (mode 0: over
 * the samples; mode 1: the Gaussian integral).
 * k_samples: [L][H][n_samples][d] post-RoPE keys; v_samples: same shape, values.                        */
int tq_calibrate_host(const tq_shape *shape, int32_t mode, const float *k_samples, const float *v_samples,
                      int64_t n_samples, uint64_t seed, tq_params *out_host);

/* ---- (a) quantize-and-pack, prefill form [PAPER.md:111-116; §3.3; §3.4; §4.2] ----------------------
 * k, v: DEVICE, [B][H][n_tokens][d] contiguous, dtype dt, pre-RoPE keys and values of layer `layer`.
 * Token i of the call is cached at index start_pos + i and its RoPE position is that index.
 * Sets seq_len[layer][b] = start_pos + n_tokens for every b.  n_tokens == 0 only sets seq_len.
 * TQ_ERR_CAPACITY if start_pos + n_tokens > max_seq.                                                    */
int tq_quantize_pack(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer,
                     const void *k, const void *v, tq_dtype dt, int32_t n_tokens, int32_t start_pos,
                     void *cuda_stream);

/* ---- (a) quantize-and-pack, per appended token [BASELINE.json:configs[2]] --------------------------
 * k, v: DEVICE, [B][H][d].  For every b the token is cached at index seq_len[layer][b] (read on the
 * device), RoPE position = that index; afterwards seq_len[layer][b] += 1 on the device.  A batch entry
 * whose cache is full is left unchanged and the cache's sticky status word is set to TQ_ERR_CAPACITY.    */
int tq_append(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer, const void *k,
              const void *v, tq_dtype dt, void *cuda_stream);

/* ---- (b) fused decode attention [PAPER.md:118-124; Algorithm 1, 223-237; north_star] ---------------
 * Layers layer_begin .. layer_begin + n_layers_call - 1 in one call (1 for a real model).
 * q: DEVICE [n_layers_call][B][H][d], pre-RoPE queries, dtype dt.  q_pos: DEVICE int32
 * [n_layers_call][B] RoPE positions of the queries, or NULL for seq_len - 1 (the query is the newest
 * cached token).  out: DEVICE [n_layers_call][B][H][d], dtype dt.  Attends, without a mask, to all
 * seq_len[layer][b] cached tokens; an empty cache gives out = 0.  t_hint: upper bound on seq_len used
 * only to size the split-K grid (0 = max_seq).  workspace: see tq_decode_workspace_bytes.               */
int tq_decode_attn(const tq_shape *shape, const tq_params *dev, const tq_cache *cache, int32_t layer_begin,
                   int32_t n_layers_call, const void *q, const int32_t *q_pos, tq_dtype dt, void *out,
                   int32_t t_hint, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- (b) fused decode attention for callers that cannot allocate device memory -------------------------------------
 * Who this is for.  tq_decode_attn needs a workspace, and somebody has to cudaMalloc it.  Some callers cannot: a
 * plug-in living inside a host application whose memory pool owns the whole device and hands out input and output
 * tensors only; code that runs where an allocation is forbidden because cudaMalloc synchronises the device (a serving
 * loop with a latency budget, a callback of somebody else's runtime); a process started with every byte of HBM already
 * handed to other tenants.  For them the library carries its own workspace: a zero-initialised array of
 * TQ_NOALLOC_SCRATCH_BYTES (24 MiB) in device global memory, part of the library image.  Every GPU on which the
 * process uses the library holds those 24 MiB from the moment the library's device code is loaded there until the
 * process exits, whether this entry point is ever called or not.
 *
 * What it computes: exactly tq_decode_attn (same arguments minus workspace / workspace_bytes, same kernels, same
 * validation and status codes, same results); the split-K partials, query operands, dequantisation tables and arrival
 * counters live in the built-in array.  The caller still owns and passes q, q_pos, out, the cache and the calibration
 * arrays.  The call performs no cudaMalloc / cudaFree and calls no routine that allocates; it enqueues one small
 * cudaMemsetAsync (the arrival counters, which must start at zero) and the two kernels on cuda_stream.
 *
 * Limit: tq_decode_workspace_bytes(shape, n_layers_call) must not exceed TQ_NOALLOC_SCRATCH_BYTES, otherwise the
 * call returns TQ_ERR_CAPACITY and launches nothing (tq_noalloc_scratch_bytes() returns the limit at run time).
 * 24 MiB covers every configuration of BASELINE.json, v_qjl = 1 and all 33 layers of configs[1] in one call
 * included (22.3 MiB); ask for fewer layers per call when a shape does not fit.
 *
 * First call on each device: the library looks up the device address of the array (cudaGetSymbolAddress, once per
 * device, with that device current) and remembers it.  Make that first call outside any stream capture — e.g. one
 * warm-up call at start-up on every device the thread will use.
 *
 * Sharing: there is ONE array per device and every call on that device uses it, with whatever the previous call left
 * in it (the entry point clears the only part that has to start at zero).  Two such calls that can overlap on the
 * GPU — different streams without an event between them, or two host threads — race on it and give wrong results:
 * keep the calls of one device on one stream, or order them with events.  tq_decode_attn with a caller-owned
 * workspace has no such restriction across workspaces and stays the entry point for everybody who can allocate.    */
#define TQ_NOALLOC_SCRATCH_BYTES (24u << 20)
size_t tq_noalloc_scratch_bytes(void);
int tq_decode_attn_noalloc(const tq_shape *shape, const tq_params *dev, const tq_cache *cache, int32_t layer_begin,
                           int32_t n_layers_call, const void *q, const int32_t *q_pos, tq_dtype dt, void *out,
                           int32_t t_hint, void *cuda_stream);

/* ---- one decode step of one layer, fused: tq_append(k, v) followed by tq_decode_attn(q) with the query at
 * the newly appended position, in two kernel launches instead of three (the append and the query
 * preparation share one kernel and its two small tensor-core products).  q, k, v, out: DEVICE [B][H][d], dtype dt.
 * Result and cache state are identical to calling the two entry points one after the other
 * (BASELINE.json:configs[2] "each step appending one quantized token per head via tq_append").            */
int tq_decode_step(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer, const void *q,
                   const void *k, const void *v, tq_dtype dt, void *out, int32_t t_hint, void *workspace,
                   size_t workspace_bytes, void *cuda_stream);

/* ---- format conversion (tests, interchange; not hot) -----------------------------------------------
 * Canonical planes are DEVICE arrays for ONE layer, index [b][h][t] with t < n_tokens:
 * k_codes/v_codes 3d/8 bytes per entry, k_signs m/8 bytes, norms uint16.  Export reads tokens
 * 0 .. n_tokens-1 of `layer`; import writes them and sets seq_len[layer][b] = n_tokens.                  */
typedef struct {
  uint8_t *k_codes, *k_signs;
  uint16_t *k_norm, *k_rnorm;
  uint8_t *v_codes;
  uint16_t *v_norm;
  uint8_t *v_signs;  /* v_qjl = 1 only (else ignored, may be NULL): m/8 bytes per entry, like k_signs */
  uint16_t *v_rnorm; /* v_qjl = 1 only: binary16 |r_v|                                                */
} tq_canonical;

int tq_cache_export_canonical(const tq_shape *shape, const tq_cache *cache, int32_t layer, int32_t n_tokens,
                              tq_canonical *out_dev, void *cuda_stream);
int tq_cache_import_canonical(const tq_shape *shape, tq_cache *cache, int32_t layer, int32_t n_tokens,
                              const tq_canonical *in_dev, void *cuda_stream);

/* ---- host-buffer convenience (the end-to-end path bench.py times as "e2e") -------------------------
 * One decode step for one layer with HOST q/k/v/out ([B][H][d], dtype dt): copies k, v, q to the device
 * staging buffers, runs tq_decode_step, copies out back and synchronises the stream.
 * staging: DEVICE buffer of tq_step_staging_bytes() bytes.                                              */
size_t tq_step_staging_bytes(const tq_shape *shape, tq_dtype dt);
int tq_decode_step_host(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer,
                        const void *q_host, const void *k_host, const void *v_host, tq_dtype dt,
                        void *out_host, int32_t t_hint, void *staging, void *workspace,
                        size_t workspace_bytes, void *cuda_stream);

/* One decode step of n_layers_call consecutive layers with HOST buffers (the end-to-end path bench.py times as
 * "e2e"): q/k/v/out are HOST [n_layers_call][B][H][d]; three host-to-device copies, tq_decode_model_step,
 * one device-to-host copy, one stream synchronisation.  workspace: for n_layers_call layers.  staging: DEVICE, tq_model_step_staging_bytes() bytes,
 * 256-byte aligned.  Per-layer results are identical to tq_decode_step_host called layer by layer.             */
size_t tq_model_step_staging_bytes(const tq_shape *shape, tq_dtype dt, int32_t n_layers_call);
int tq_decode_model_step_host(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer_begin,
                              int32_t n_layers_call, const void *q_host, const void *k_host, const void *v_host,
                              tq_dtype dt, void *out_host, int32_t t_hint, void *staging, void *workspace,
                              size_t workspace_bytes, void *cuda_stream);

/* ---- stepper: one decode step of a run of layers captured ONCE as a CUDA graph (the serving loop's form of the step;
 * bench.py times it with host buffers as "e2e") [BASELINE.json:configs[2] "100 consecutive decode steps"; SURVEY.md §7
 * hard part 2].  tq_host_stepper_create records, for FIXED buffers q/k/v/out ([n_layers_call][B][H][d], dtype dt, valid
 * until destroy), a graph with several branches; the layers are cut into n_chunks runs of growing length (0 = the
 * library's choice):
 *   copy     : per run, the host-to-device copies of k, v, q, back to back;
 *   prep     : per run, the append + query-prep kernel behind that run's copies;
 *   main x 2 : the streaming kernels of all layers; the chains of consecutive runs alternate between two branches, so the
 *              first kernel of a run waits only for that run's prep kernel;
 *   copy-out : per group of six layers, the PI_V^T finish kernel, then the device-to-host copy of out.
 * buffers_on_host = 1: q/k/v/out are HOST buffers and must be page-locked (cudaHostAlloc / cudaHostRegister); staging is a
 * DEVICE buffer of tq_model_step_staging_bytes() bytes, 256-byte aligned.  buffers_on_host = 0: they are DEVICE buffers,
 * no copies are recorded and staging may be NULL.  workspace: tq_decode_workspace_bytes(shape, n_layers_call), zero-filled
 * once; staging and workspace are owned by the caller and used by every run.  Results and cache state are identical to
 * tq_decode_model_step(_host).  The stepper is the only object the library ever allocates (a graph and its executable, on
 * the host); create and destroy are not hot.
 * tq_host_stepper_launch: one graph launch on cuda_stream, asynchronous.  tq_host_stepper_run: launch + one stream
 * synchronisation (the caller writes this step's q/k/v into the buffers before, reads out after).  seq_len lives on the
 * device, so the same graph serves every step.  Errors: TQ_ERR_INVALID_ARG (NULL / misaligned), TQ_ERR_CAPACITY
 * (workspace), TQ_ERR_CUDA (capture failed, e.g. pageable host memory).                                                */
typedef struct tq_host_stepper tq_host_stepper;
int tq_host_stepper_create(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer_begin,
                           int32_t n_layers_call, const void *q_buf, const void *k_buf, const void *v_buf, void *out_buf,
                           int32_t buffers_on_host, tq_dtype dt, int32_t t_hint, void *staging, void *workspace,
                           size_t workspace_bytes, int32_t n_chunks, tq_host_stepper **out_stepper);
int tq_host_stepper_launch(tq_host_stepper *stepper, void *cuda_stream);
int tq_host_stepper_run(tq_host_stepper *stepper, void *cuda_stream);
int tq_host_stepper_destroy(tq_host_stepper *stepper);

/* ---- one decode step of a run of layers, DEVICE buffers [BASELINE.json:configs[2]; configs[1] for the shape] --------
 * q, k, v, out: DEVICE [n_layers_call][B][H][d], dtype dt.  Result and cache state are identical to tq_decode_step
 * called layer by layer (layers are independent: "each (layer, head)").  What differs is the launch
 * plan: ONE kernel appends the new token and prepares the query operands of every layer, then one streaming kernel
 * per layer cache is launched as a programmatic-dependent-launch chain in which only the first waits for the prep
 * kernel; the others run ahead, so that the ramp and the tail of consecutive layers overlap.  The caller must have
 * every layer's q/k/v ready before the call (a model that produces layer l+1's inputs from layer l's output uses
 * tq_decode_step).  workspace: tq_decode_workspace_bytes(shape, n_layers_call), zero-filled once.                  */
int tq_decode_model_step(const tq_shape *shape, const tq_params *dev, tq_cache *cache, int32_t layer_begin,
                         int32_t n_layers_call, const void *q, const void *k, const void *v, tq_dtype dt, void *out,
                         int32_t t_hint, void *workspace, size_t workspace_bytes, void *cuda_stream);

const char *tq_status_string(int status);
/* Number of kernels the library launched since load (bench.py's gpu_launches).                          */
int64_t tq_launch_count(void);
/* ---- measurement and test hooks: compiled ONLY with -DTQ_TEST_HOOKS ------------------------------------------------
 * The three functions below, and the fp32 CUDA-core cross-check kernel behind the last of them, exist only in a library
 * built with -DTQ_TEST_HOOKS.  That is the build the tests, bench.py and __graft_entry__ use
 * (`python -m paper_2603_26110_b200.build`, the default).  `python -m paper_2603_26110_b200.build --product` leaves them
 * out: that library exports none of the three symbols and its product path reads no process-wide switch.            */
#ifdef TQ_TEST_HOOKS
/* Measurement hook, NOT part of the product path (bench.py's roofline leg and one test use it): while on,
 * tq_decode_attn / tq_decode_model_step skip the append + query-prep kernel and re-use the query operands their
 * previous ordinary call left in the workspace (same queries, same layers), so that a run of such calls times
 * the streaming kernel alone.  Process-wide (an atomic flag); results are only meaningful directly after an
 * ordinary call with the same arguments; always switch it off again.  on = 2: tq_decode_model_step also leaves out its
 * finish kernel (the streaming launches alone; the outputs are then not written).                          */
void tq_profile_decode_main_only(int on);
/* Test / sweep knobs (process-wide, not part of the product path; both default to 0 = the library's own choice):
 * CTAs per unit of the streaming decode kernel; 1 = route tq_quantize_pack to the fp32 CUDA-core cross-check kernel.
 * That kernel implements the default mode only: with residual_mode = 1 or v_qjl = 1 the setting is ignored and the
 * tensor-core kernel runs.                                                                                            */
void tq_debug_set_decode_nsplit(int nsplit);
void tq_debug_set_quantize_impl(int fp32_cuda_cores);
#endif /* TQ_TEST_HOOKS */

#ifdef __cplusplus
}
#endif
#endif /* TQ_H_ */
