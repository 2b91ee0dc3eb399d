// tq_api.cu — the extern "C" boundary declared in include/tq.h: host-side validation, size arithmetic,
// launch configuration.  No torch types, no allocation, no hidden synchronisation (except the explicit
// host-buffer convenience call tq_decode_step_host, which must synchronise to hand back host data).
#include <atomic>
#include <cstring>

#include "tq_common.cuh"

namespace tq {

static std::atomic<long long> g_launches{0};
// Measurement / test hooks exist only in builds with -DTQ_TEST_HOOKS (what the tests and bench.py build; include/tq.h).
// Without it the three values below are compile-time zeros and the product path carries no mutable process-wide state.
#ifdef TQ_TEST_HOOKS
static std::atomic<int> g_profile_skip_prep{0};  // tq_profile_decode_main_only (a setter may run on another thread)
static std::atomic<int> g_debug_nsplit{0};       // tq_debug_set_decode_nsplit
static int profile_skip_prep() { return g_profile_skip_prep.load(std::memory_order_relaxed); }
static int debug_nsplit() { return g_debug_nsplit.load(std::memory_order_relaxed); }
#else
static constexpr int profile_skip_prep() { return 0; }
static constexpr int debug_nsplit() { return 0; }
#endif
// Launches recorded into a stream capture are not launches yet: while the stepper captures (thread-local capture mode,
// so every recorded launch comes from this thread) they are counted apart and added at every replay.
static thread_local bool t_capturing = false;
static thread_local int t_captured = 0;
void count_launch(int n) {
  if (t_capturing)
    t_captured += n;
  else
    g_launches.fetch_add(n, std::memory_order_relaxed);
}


constexpr int kMaxSplits = 64;  // = kMaxSegments in tq_decode.cu

// Splits per unit for the streaming decode kernel.  Model: CTAs land round-robin on the SMs and the CTAs of an
// SM share it, so the launch takes (max CTAs on one SM) x (tiles per CTA + a fixed per-CTA cost for the table
// build, the cross-warp reduction and the split-K hand-off, in tile units).
static int choose_nsplit(int units, int ntiles, int sms) {
  const double kFixedTiles = 3.0;
  int best = 1;
  double best_t = 1e300;
  for (int ns = 1; ns <= kMaxSplits && (ns == 1 || ntiles / ns >= 4); ++ns) {
    const long ctas = (long)units * ns;
    const long per_sm = (ctas + sms - 1) / sms;
    const int per = (ntiles + ns - 1) / ns;
    const double t = (double)per_sm * (per + kFixedTiles + (ns > 1 ? 1.0 : 0.0));
    if (t < best_t * 0.97) {  // prefer fewer splits unless the gain is real
      best_t = t;
      best = ns;
    }
  }
  return best;
}

// split factor of a launch: the plan above, or the value set with tq_debug_set_decode_nsplit (tests, sweeps)
static int pick_nsplit(int units, int ntiles, int sms) {
  const int forced = debug_nsplit();
  return forced >= 1 && forced <= kMaxSplits ? forced : choose_nsplit(units, ntiles, sms);
}

// SM count of the CURRENT device (a process may drive several): cached per device ordinal
static int num_sms() {
  constexpr int kMaxDev = 64;
  static std::atomic<int> cached[kMaxDev];  // zero-initialised: 0 = not queried yet
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -1;
  if (dev >= 0 && dev < kMaxDev && (n = cached[dev].load(std::memory_order_relaxed)) > 0) return n;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return -1;
  if (dev >= 0 && dev < kMaxDev) cached[dev].store(n, std::memory_order_relaxed);
  return n;
}

static int check_shape(const tq_shape* s, CacheGeom* g) {
  if (!s) return TQ_ERR_INVALID_ARG;
  if (s->n_layers <= 0 || s->batch <= 0 || s->n_heads <= 0 || s->max_seq <= 0 || !(s->rope_base > 0.f))
    return TQ_ERR_INVALID_ARG;
  if (s->rope_layout != 0 && s->rope_layout != 1) return TQ_ERR_INVALID_ARG;
  if (s->residual_mode != 0 && s->residual_mode != 1) return TQ_ERR_INVALID_ARG;
  if (s->v_qjl != 0 && s->v_qjl != 1) return TQ_ERR_INVALID_ARG;
  if ((s->head_dim != 64 && s->head_dim != 128) || s->qjl_dim != s->head_dim || (s->v_qjl == 1 && s->residual_mode == 1))
    return TQ_ERR_UNSUPPORTED;
  if (!make_geom(s, g)) return TQ_ERR_INVALID_ARG;
  return TQ_OK;
}

static bool aligned16(const void* p) { return p && ((uintptr_t)p & 15u) == 0; }

static int check_params(const tq_params* p, const tq_shape* s) {
  if (!p) return TQ_ERR_INVALID_ARG;
  if (s->residual_mode == 1 && (!p->ebar_k || ((uintptr_t)p->ebar_k & 3u))) return TQ_ERR_INVALID_ARG;
  if (!aligned16(p->pi_k) || !aligned16(p->pi_v) || !aligned16(p->lut_k) || !aligned16(p->lut_v) || !aligned16(p->S) ||
      !aligned16(p->rope_cs))
    return TQ_ERR_INVALID_ARG;
  return TQ_OK;
}

struct WorkspaceGeom {
  size_t off_counters, off_frags, off_tabs, off_orot, off_partials, total;
  size_t frag_words;
  size_t rec;  // floats per split-K partial record
};
static WorkspaceGeom workspace_geom(const CacheGeom& g, int n_layers_call) {
  WorkspaceGeom w;
  size_t units = (size_t)n_layers_call * g.B * g.H;
  w.off_counters = 0;
  w.frag_words = g.D == 64 ? FragLayout<64>::kWords : FragLayout<128>::kWords;
  w.off_frags = (units * 4 + 255) / 256 * 256;
  w.off_tabs = w.off_frags + (units * w.frag_words * 4 + 255) / 256 * 256;
  w.off_orot = w.off_tabs + ((size_t)n_layers_call * g.H * kTabWords * 4 + 255) / 256 * 256;
  w.off_partials = w.off_orot + (units * g.D * 4 + 255) / 256 * 256;
  w.rec = (size_t)decode_record_floats(g.D, g.vq != 0);
  w.total = w.off_partials + units * kMaxSplits * w.rec * 4;
  return w;
}

}  // namespace tq

using namespace tq;

extern "C" {

size_t tq_cache_bytes(const tq_shape* shape) {
  CacheGeom g;
  return check_shape(shape, &g) == TQ_OK ? g.total_bytes : 0;
}
size_t tq_cache_bytes_per_token_head(const tq_shape* shape) {
  CacheGeom g;
  return check_shape(shape, &g) == TQ_OK ? (g.tile_bytes + g.vsk_tile_bytes) / kTile : 0;
}
size_t tq_cache_seq_len_offset(const tq_shape* shape) {
  CacheGeom g;
  return check_shape(shape, &g) == TQ_OK ? g.off_seq_len : 0;
}
size_t tq_cache_status_offset(const tq_shape* shape) {
  CacheGeom g;
  return check_shape(shape, &g) == TQ_OK ? g.off_status : 0;
}
size_t tq_decode_workspace_bytes(const tq_shape* shape, int32_t n_layers_call) {
  CacheGeom g;
  if (check_shape(shape, &g) != TQ_OK || n_layers_call <= 0 || n_layers_call > g.L) return 0;
  return workspace_geom(g, n_layers_call).total;
}
size_t tq_canonical_plane_bytes(const tq_shape* shape, int32_t plane, int32_t n_tokens) {
  CacheGeom g;
  if (check_shape(shape, &g) != TQ_OK || n_tokens < 0) return 0;
  size_t e = (size_t)g.B * g.H * n_tokens;
  switch (plane) {
    case 0:
    case 4:
      return e * (3 * g.D / 8);
    case 1:
      return e * (g.D / 8);
    case 6:
      return g.vq ? e * (g.D / 8) : 0;
    case 2:
    case 3:
    case 5:
      return e * 2;
    case 7:
      return g.vq ? e * 2 : 0;
    default:
      return 0;
  }
}

int tq_quantize_pack(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer, const void* k,
                     const void* v, tq_dtype dt, int32_t n_tokens, int32_t start_pos, void* cuda_stream) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if ((rc = check_params(dev, shape)) != TQ_OK) return rc;
  if (!cache || !cache->data || ((uintptr_t)cache->data & 255u)) return TQ_ERR_INVALID_ARG;
  if (layer < 0 || layer >= g.L || n_tokens < 0 || start_pos < 0) return TQ_ERR_INVALID_ARG;
  if (dt != TQ_F16 && dt != TQ_F32) return TQ_ERR_INVALID_ARG;
  if (n_tokens > 0 && (!aligned16(k) || !aligned16(v))) return TQ_ERR_INVALID_ARG;
  if ((long long)start_pos + n_tokens > g.max_seq) return TQ_ERR_CAPACITY;
  int sms = num_sms();
  if (sms <= 0) return TQ_ERR_CUDA;
  QuantArgs a;
  a.cv = make_view(g, cache->data);
  a.k = k;
  a.v = v;
  a.pi_k = dev->pi_k + (size_t)layer * g.H * g.D * g.D;
  a.pi_v = dev->pi_v + (size_t)layer * g.H * g.D * g.D;
  a.lut_k = dev->lut_k + (size_t)layer * g.H * 8;
  a.lut_v = dev->lut_v + (size_t)layer * g.H * 8;
  a.S = dev->S;
  a.rope_cs = dev->rope_cs;
  a.layer = layer;
  a.n_tokens = n_tokens;
  a.start_pos = start_pos;
  a.rope_layout = shape->rope_layout;
  a.tiles_per_cta = 1;
  a.literal = shape->residual_mode == 1;
  a.ebar_k = a.literal ? dev->ebar_k + (size_t)layer * g.H : nullptr;
  return launch_quantize_pack(a, g.D, dt, sms, (cudaStream_t)cuda_stream) == cudaSuccess ? TQ_OK : TQ_ERR_CUDA;
}

// Shared body of tq_append / tq_decode_attn / tq_decode_step: validation, then
// [prep kernel (append and/or query prep)] + [streaming decode kernel].
static int run_decode(const tq_shape* shape, const tq_params* dev, const tq_cache* cache, int32_t layer_begin,
                      int32_t n_layers_call, const void* q, const void* k, const void* v, const int32_t* q_pos,
                      tq_dtype dt, void* out, int32_t t_hint, void* workspace, size_t workspace_bytes, bool do_append,
                      bool do_query, void* cuda_stream) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if ((rc = check_params(dev, shape)) != TQ_OK) return rc;
  if (!cache || !cache->data || ((uintptr_t)cache->data & 255u)) return TQ_ERR_INVALID_ARG;
  if (layer_begin < 0 || n_layers_call <= 0 || layer_begin + n_layers_call > g.L) return TQ_ERR_INVALID_ARG;
  if (dt != TQ_F16 && dt != TQ_F32) return TQ_ERR_INVALID_ARG;
  if (do_append && (!aligned16(k) || !aligned16(v))) return TQ_ERR_INVALID_ARG;
  WorkspaceGeom w = workspace_geom(g, n_layers_call);
  if (do_query) {
    if (!aligned16(q) || !aligned16(out) || !workspace || ((uintptr_t)workspace & 255u)) return TQ_ERR_INVALID_ARG;
    if (t_hint < 0) return TQ_ERR_INVALID_ARG;
    if (workspace_bytes < w.total) return TQ_ERR_CAPACITY;
  }
  const int sms = num_sms();
  if (sms <= 0) return TQ_ERR_CUDA;
  const int th = (t_hint == 0 || t_hint > g.max_seq) ? g.max_seq : t_hint;
  const int ntiles = (th + kTile - 1) / kTile;
  const int nsplit = pick_nsplit(n_layers_call * g.B * g.H, ntiles, sms);
  unsigned char* ws = (unsigned char*)workspace;
  DecodeArgs a;
  a.cv = make_view(g, cache->data);
  a.pi_k = dev->pi_k;
  a.pi_v = dev->pi_v;
  a.lut_k = dev->lut_k;
  a.lut_v = dev->lut_v;
  a.S = dev->S;
  a.rope_cs = dev->rope_cs;
  a.q = q;
  a.out = out;
  a.q_pos = q_pos;
  a.counters = ws ? (int*)(ws + w.off_counters) : nullptr;
  a.frags = ws ? (unsigned*)(ws + w.off_frags) : nullptr;
  a.tabs = ws ? (unsigned*)(ws + w.off_tabs) : nullptr;
  a.orot = nullptr;
  a.partials = ws ? (float*)(ws + w.off_partials) : nullptr;
  a.layer_begin = layer_begin;
  a.n_layers_call = n_layers_call;
  a.nsplit = nsplit;
  a.per = (ntiles + nsplit - 1) / nsplit;
  a.chain_mode = 0;
  a.rope_layout = shape->rope_layout;
  a.dt = (int)dt;
  a.literal = shape->residual_mode == 1;
  a.ebar_k = a.literal ? dev->ebar_k : nullptr;
  // one prep launch (append and / or query operands of every layer of the call), then one streaming launch over all units
  if (!(profile_skip_prep() && do_query && !do_append) &&
      launch_prep(a, k, v, g.D, sms, do_append, do_query, (cudaStream_t)cuda_stream) != cudaSuccess)
    return TQ_ERR_CUDA;
  if (do_query && launch_decode(a, g.D, true, (cudaStream_t)cuda_stream) != cudaSuccess) return TQ_ERR_CUDA;
  return TQ_OK;
}

int tq_append(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer, const void* k, const void* v,
              tq_dtype dt, void* cuda_stream) {
  return run_decode(shape, dev, cache, layer, 1, nullptr, k, v, nullptr, dt, nullptr, 0, nullptr, 0, true, false,
                    cuda_stream);
}

int tq_decode_attn(const tq_shape* shape, const tq_params* dev, const tq_cache* cache, int32_t layer_begin,
                   int32_t n_layers_call, const void* q, const int32_t* q_pos, tq_dtype dt, void* out, int32_t t_hint,
                   void* workspace, size_t workspace_bytes, void* cuda_stream) {
  return run_decode(shape, dev, cache, layer_begin, n_layers_call, q, nullptr, nullptr, q_pos, dt, out, t_hint, workspace,
                    workspace_bytes, false, true, cuda_stream);
}

}  // extern "C"

// ---- tq_decode_attn_noalloc: the decode workspace inside the library image (include/tq.h says for whom) -------------
// The array below is the workspace of tq_decode_attn for callers that cannot cudaMalloc one.  In HOST code its name is
// only a handle for the runtime, never a pointer a kernel may be given: the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current, and is remembered per device ordinal (every
// device has its own copy of the array at its own address).
namespace tq {
static __device__ __align__(256) unsigned char g_noalloc_scratch[TQ_NOALLOC_SCRATCH_BYTES];

static int noalloc_scratch_address(unsigned char** out) {
  constexpr int kMaxDev = 64;
  static std::atomic<unsigned char*> cached[kMaxDev];  // zero-initialised: nullptr = not asked yet on that device
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return TQ_ERR_CUDA;
  const bool slot = dev >= 0 && dev < kMaxDev;
  unsigned char* p = slot ? cached[dev].load(std::memory_order_acquire) : nullptr;
  if (!p) {  // set-up of this device (two threads may both ask: they get the same answer)
    if (cudaGetSymbolAddress((void**)&p, g_noalloc_scratch) != cudaSuccess || !p) {
      cudaGetLastError();
      return TQ_ERR_CUDA;
    }
    if (slot) cached[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return TQ_OK;
}
}  // namespace tq

extern "C" {

size_t tq_noalloc_scratch_bytes(void) { return (size_t)TQ_NOALLOC_SCRATCH_BYTES; }

int tq_decode_attn_noalloc(const tq_shape* shape, const tq_params* dev, const tq_cache* cache, int32_t layer_begin,
                           int32_t n_layers_call, const void* q, const int32_t* q_pos, tq_dtype dt, void* out,
                           int32_t t_hint, void* cuda_stream) {
  // shape and layer count first (the size check needs them), with tq_decode_attn's own status codes; every other
  // argument is checked by the shared validation of run_decode below, which launches nothing on an error
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if (n_layers_call <= 0 || n_layers_call > g.L) return TQ_ERR_INVALID_ARG;
  const WorkspaceGeom w = workspace_geom(g, n_layers_call);
  if (w.total > (size_t)TQ_NOALLOC_SCRATCH_BYTES) return TQ_ERR_CAPACITY;  // the built-in array is too small: fewer layers per call
  unsigned char* scratch = nullptr;
  if ((rc = noalloc_scratch_address(&scratch)) != TQ_OK) return rc;
  // The array keeps what the last call left there, possibly a call of another shape whose query operands or partials
  // lie where this call's split-K arrival counters are: those must start at zero (nothing else is read before this
  // call's own kernels have written it)
  if (cudaMemsetAsync(scratch + w.off_counters, 0, w.off_frags - w.off_counters, (cudaStream_t)cuda_stream) != cudaSuccess)
    return TQ_ERR_CUDA;
  return run_decode(shape, dev, cache, layer_begin, n_layers_call, q, nullptr, nullptr, q_pos, dt, out, t_hint, scratch,
                    (size_t)TQ_NOALLOC_SCRATCH_BYTES, false, true, cuda_stream);
}

int tq_decode_step(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer, const void* q,
                   const void* k, const void* v, tq_dtype dt, void* out, int32_t t_hint, void* workspace,
                   size_t workspace_bytes, void* cuda_stream) {
  return run_decode(shape, dev, cache, layer, 1, q, k, v, nullptr, dt, out, t_hint, workspace, workspace_bytes, true,
                    true, cuda_stream);
}

int tq_cache_export_canonical(const tq_shape* shape, const tq_cache* cache, int32_t layer, int32_t n_tokens,
                              tq_canonical* out_dev, void* cuda_stream) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if (!cache || !cache->data || !out_dev || layer < 0 || layer >= g.L || n_tokens < 0) return TQ_ERR_INVALID_ARG;
  if (n_tokens > g.max_seq) return TQ_ERR_CAPACITY;
  if (n_tokens > 0 && (!out_dev->k_codes || !out_dev->k_signs || !out_dev->k_norm || !out_dev->k_rnorm ||
                       !out_dev->v_codes || !out_dev->v_norm || (g.vq && (!out_dev->v_signs || !out_dev->v_rnorm))))
    return TQ_ERR_INVALID_ARG;
  if (num_sms() <= 0) return TQ_ERR_CUDA;
  return launch_export(g, make_view(g, cache->data), layer, n_tokens, *out_dev, (cudaStream_t)cuda_stream) == cudaSuccess
             ? TQ_OK
             : TQ_ERR_CUDA;
}

int tq_cache_import_canonical(const tq_shape* shape, tq_cache* cache, int32_t layer, int32_t n_tokens,
                              const tq_canonical* in_dev, void* cuda_stream) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if (!cache || !cache->data || !in_dev || layer < 0 || layer >= g.L || n_tokens < 0) return TQ_ERR_INVALID_ARG;
  if (n_tokens > g.max_seq) return TQ_ERR_CAPACITY;
  if (n_tokens > 0 && (!in_dev->k_codes || !in_dev->k_signs || !in_dev->k_norm || !in_dev->k_rnorm || !in_dev->v_codes ||
                       !in_dev->v_norm || (g.vq && (!in_dev->v_signs || !in_dev->v_rnorm))))
    return TQ_ERR_INVALID_ARG;
  if (num_sms() <= 0) return TQ_ERR_CUDA;
  return launch_import(g, make_view(g, cache->data), layer, n_tokens, *in_dev, (cudaStream_t)cuda_stream) == cudaSuccess
             ? TQ_OK
             : TQ_ERR_CUDA;
}

// Validated launch plan of one model decode step (tq_decode_model_step and the host stepper share it).
struct ModelStepPlan {
  CacheGeom g;
  WorkspaceGeom w;
  DecodeArgs a;  // the whole call: layers [layer_begin, layer_begin + n_layers_call)
  const unsigned char *k, *v;
  size_t esz;
  int sms;
};

static int plan_model_step(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer_begin,
                           int32_t n_layers_call, const void* q, const void* k, const void* v, tq_dtype dt, void* out,
                           int32_t t_hint, void* workspace, size_t workspace_bytes, ModelStepPlan* p) {
  CacheGeom& g = p->g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if ((rc = check_params(dev, shape)) != TQ_OK) return rc;
  if (!cache || !cache->data || ((uintptr_t)cache->data & 255u)) return TQ_ERR_INVALID_ARG;
  if (layer_begin < 0 || n_layers_call <= 0 || layer_begin + n_layers_call > g.L) return TQ_ERR_INVALID_ARG;
  if (dt != TQ_F16 && dt != TQ_F32) return TQ_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out) || !workspace || ((uintptr_t)workspace & 255u))
    return TQ_ERR_INVALID_ARG;
  if (t_hint < 0) return TQ_ERR_INVALID_ARG;
  p->w = workspace_geom(g, n_layers_call);
  if (workspace_bytes < p->w.total) return TQ_ERR_CAPACITY;
  p->sms = num_sms();
  if (p->sms <= 0) return TQ_ERR_CUDA;
  const int th = (t_hint == 0 || t_hint > g.max_seq) ? g.max_seq : t_hint;
  const int ntiles = (th + kTile - 1) / kTile;
  const int nsplit = pick_nsplit(g.B * g.H, ntiles, p->sms);
  p->esz = dt == TQ_F16 ? 2 : 4;
  p->k = (const unsigned char*)k, p->v = (const unsigned char*)v;
  unsigned char* ws = (unsigned char*)workspace;
  DecodeArgs& a = p->a;
  a.cv = make_view(g, cache->data);
  a.pi_k = dev->pi_k, a.pi_v = dev->pi_v, a.lut_k = dev->lut_k, a.lut_v = dev->lut_v, a.S = dev->S, a.rope_cs = dev->rope_cs;
  a.q = q, a.out = out, a.q_pos = nullptr;
  a.counters = (int*)(ws + p->w.off_counters);
  a.frags = (unsigned*)(ws + p->w.off_frags);
  a.tabs = (unsigned*)(ws + p->w.off_tabs);
  a.orot = (float*)(ws + p->w.off_orot);
  a.partials = (float*)(ws + p->w.off_partials);
  a.layer_begin = layer_begin, a.n_layers_call = n_layers_call;
  a.nsplit = nsplit, a.per = (ntiles + nsplit - 1) / nsplit;
  a.chain_mode = 0, a.rope_layout = shape->rope_layout, a.dt = (int)dt;
  a.literal = shape->residual_mode == 1;
  a.ebar_k = a.literal ? dev->ebar_k : nullptr;
  return TQ_OK;
}

// the arguments of layers [l0, l0 + nl) of the planned call (every pointer advanced to that sub-range)
static DecodeArgs sub_args(const ModelStepPlan& p, int l0, int nl) {
  DecodeArgs b = p.a;
  const size_t u0 = (size_t)l0 * p.g.B * p.g.H;
  b.q = (const unsigned char*)p.a.q + u0 * p.g.D * p.esz;
  b.out = (unsigned char*)p.a.out + u0 * p.g.D * p.esz;
  b.counters = p.a.counters + u0;
  b.frags = p.a.frags + u0 * p.w.frag_words;
  b.tabs = p.a.tabs + (size_t)l0 * p.g.H * kTabWords;
  b.orot = p.a.orot + u0 * p.g.D;
  b.partials = p.a.partials + u0 * kMaxSplits * p.w.rec;
  b.layer_begin = p.a.layer_begin + l0, b.n_layers_call = nl;
  return b;
}

int tq_decode_model_step(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer_begin,
                         int32_t n_layers_call, const void* q, const void* k, const void* v, tq_dtype dt, void* out,
                         int32_t t_hint, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  ModelStepPlan p;
  int rc = plan_model_step(shape, dev, cache, layer_begin, n_layers_call, q, k, v, dt, out, t_hint, workspace,
                           workspace_bytes, &p);
  if (rc != TQ_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // one prep launch for every layer of the step (append + query operands), then one streaming launch per layer cache:
  // the first waits for the prep kernel, the others run ahead of one another (DecodeArgs::chain_mode); they leave o'/l
  // in the workspace and one last launch applies PI_V^T to every unit of the step
  const int hook = profile_skip_prep();  // measurement hook, always 0 without TQ_TEST_HOOKS
  if (!hook && launch_prep(p.a, p.k, p.v, p.g.D, p.sms, true, true, st) != cudaSuccess) return TQ_ERR_CUDA;
  for (int l = 0; l < n_layers_call; ++l) {
    DecodeArgs b = sub_args(p, l, 1);
    b.chain_mode = l == 0 ? 0 : 1;
    if (launch_decode(b, p.g.D, false, st) != cudaSuccess) return TQ_ERR_CUDA;
  }
  // (measurement hook level 2: the streaming launches alone, without the finish kernel)
  if (hook != 2 && launch_finish(p.a, p.g.D, true, st) != cudaSuccess) return TQ_ERR_CUDA;
  return TQ_OK;
}

size_t tq_step_staging_bytes(const tq_shape* shape, tq_dtype dt) {
  CacheGeom g;
  if (check_shape(shape, &g) != TQ_OK) return 0;
  size_t vec = ((size_t)g.B * g.H * g.D * (dt == TQ_F16 ? 2 : 4) + 255) / 256 * 256;
  return 4 * vec;
}

int tq_decode_step_host(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer, const void* q_host,
                        const void* k_host, const void* v_host, tq_dtype dt, void* out_host, int32_t t_hint,
                        void* staging, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if (!q_host || !k_host || !v_host || !out_host || !staging || ((uintptr_t)staging & 255u)) return TQ_ERR_INVALID_ARG;
  if (dt != TQ_F16 && dt != TQ_F32) return TQ_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  size_t bytes = (size_t)g.B * g.H * g.D * (dt == TQ_F16 ? 2 : 4);
  size_t vec = (bytes + 255) / 256 * 256;
  unsigned char* s = (unsigned char*)staging;
  void *dq = s, *dk = s + vec, *dv = s + 2 * vec, *dout = s + 3 * vec;
  if (cudaMemcpyAsync(dk, k_host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return TQ_ERR_CUDA;
  if (cudaMemcpyAsync(dv, v_host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return TQ_ERR_CUDA;
  if (cudaMemcpyAsync(dq, q_host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return TQ_ERR_CUDA;
  if ((rc = tq_decode_step(shape, dev, cache, layer, dq, dk, dv, dt, dout, t_hint, workspace, workspace_bytes,
                           cuda_stream)) != TQ_OK)
    return rc;
  if (cudaMemcpyAsync(out_host, dout, bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return TQ_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return TQ_ERR_CUDA;
  return TQ_OK;
}

size_t tq_model_step_staging_bytes(const tq_shape* shape, tq_dtype dt, int32_t n_layers_call) {
  CacheGeom g;
  if (check_shape(shape, &g) != TQ_OK || n_layers_call <= 0 || n_layers_call > g.L) return 0;
  size_t vec = ((size_t)n_layers_call * g.B * g.H * g.D * (dt == TQ_F16 ? 2 : 4) + 255) / 256 * 256;
  return 4 * vec;
}

int tq_decode_model_step_host(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer_begin,
                              int32_t n_layers_call, const void* q_host, const void* k_host, const void* v_host,
                              tq_dtype dt, void* out_host, int32_t t_hint, void* staging, void* workspace,
                              size_t workspace_bytes, void* cuda_stream) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if (!q_host || !k_host || !v_host || !out_host || !staging || ((uintptr_t)staging & 255u)) return TQ_ERR_INVALID_ARG;
  if (dt != TQ_F16 && dt != TQ_F32) return TQ_ERR_INVALID_ARG;
  if (layer_begin < 0 || n_layers_call <= 0 || layer_begin + n_layers_call > g.L) return TQ_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t per_layer = (size_t)g.B * g.H * g.D * (dt == TQ_F16 ? 2 : 4);
  const size_t bytes = per_layer * n_layers_call;
  const size_t vec = (bytes + 255) / 256 * 256;
  unsigned char* s = (unsigned char*)staging;
  unsigned char *dq = s, *dk = s + vec, *dv = s + 2 * vec, *dout = s + 3 * vec;
  if (cudaMemcpyAsync(dk, k_host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return TQ_ERR_CUDA;
  if (cudaMemcpyAsync(dv, v_host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return TQ_ERR_CUDA;
  if (cudaMemcpyAsync(dq, q_host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return TQ_ERR_CUDA;
  if ((rc = tq_decode_model_step(shape, dev, cache, layer_begin, n_layers_call, dq, dk, dv, dt, dout, t_hint, workspace,
                                 workspace_bytes, cuda_stream)) != TQ_OK)
    return rc;
  if (cudaMemcpyAsync(out_host, dout, bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return TQ_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return TQ_ERR_CUDA;
  return TQ_OK;
}

// ---- stepper: one decode step of a run of layers captured ONCE as a CUDA graph; its branches -----------------------
//   copy      : (host buffers only) per layer chunk, the H2D copies of k, v, q, back to back
//   prep      : per chunk, the append + query-prep kernel, behind that chunk's copies
//   main, main2: the streaming kernels; the chains of consecutive chunks alternate between the two branches, so the first
//                kernel of a chunk waits for that chunk's prep kernel only (and for the chunk two in front), the others run
//                ahead as in tq_decode_model_step
//   copy-out  : per group of six layers, the finish kernel (PI_V^T), then the D2H copy of out (host buffers only)
struct tq_host_stepper {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  int n_launches = 0;  // kernels inside one replay (tq_launch_count bookkeeping)
};

int tq_host_stepper_create(const tq_shape* shape, const tq_params* dev, tq_cache* cache, int32_t layer_begin,
                           int32_t n_layers_call, const void* q_buf, const void* k_buf, const void* v_buf, void* out_buf,
                           int32_t buffers_on_host, tq_dtype dt, int32_t t_hint, void* staging, void* workspace,
                           size_t workspace_bytes, int32_t n_chunks, tq_host_stepper** out_stepper) {
  CacheGeom g;
  int rc = check_shape(shape, &g);
  if (rc != TQ_OK) return rc;
  if (!out_stepper) return TQ_ERR_INVALID_ARG;
  *out_stepper = nullptr;
  if (!q_buf || !k_buf || !v_buf || !out_buf) return TQ_ERR_INVALID_ARG;
  if (buffers_on_host && (!staging || ((uintptr_t)staging & 255u))) return TQ_ERR_INVALID_ARG;
  if (dt != TQ_F16 && dt != TQ_F32) return TQ_ERR_INVALID_ARG;
  if (layer_begin < 0 || n_layers_call <= 0 || layer_begin + n_layers_call > g.L) return TQ_ERR_INVALID_ARG;
  constexpr int kMaxChunks = 64;
  // measured at configs[2] x 33 layers (value 48.8 G token-heads/s): 2 chunks 37.6 G end to end, 3: 41.7, 4: 42.5, 6: 39.4,
  // 8: 37.4 (more chunks = more and smaller prep launches)
  if (n_chunks <= 0) n_chunks = n_layers_call >= 16 ? 4 : (n_layers_call >= 4 ? 2 : 1);
  if (n_chunks > n_layers_call) n_chunks = n_layers_call;
  if (n_chunks > kMaxChunks / 2) n_chunks = kMaxChunks / 2;
  const size_t per_layer = (size_t)g.B * g.H * g.D * (dt == TQ_F16 ? 2 : 4);
  const size_t vec = (per_layer * n_layers_call + 255) / 256 * 256;
  unsigned char* s = (unsigned char*)staging;
  const unsigned char *dq = buffers_on_host ? s : (const unsigned char*)q_buf, *dk = buffers_on_host ? s + vec : (const unsigned char*)k_buf,
                      *dv = buffers_on_host ? s + 2 * vec : (const unsigned char*)v_buf;
  unsigned char* dout = buffers_on_host ? s + 3 * vec : (unsigned char*)out_buf;
  ModelStepPlan p;
  if ((rc = plan_model_step(shape, dev, cache, layer_begin, n_layers_call, dq, dk, dv, dt, dout, t_hint, workspace,
                            workspace_bytes, &p)) != TQ_OK)
    return rc;

  cudaStream_t s_main = nullptr, s_main2 = nullptr, s_in = nullptr, s_out = nullptr, s_copy = nullptr;
  cudaEvent_t fork = nullptr, join_in = nullptr, join_out = nullptr, join_copy = nullptr, join_main2 = nullptr;
  cudaEvent_t prep_done[kMaxChunks] = {}, chain_done[kMaxChunks] = {}, copy_done[kMaxChunks] = {};
  bool ok = cudaStreamCreateWithFlags(&s_main, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&s_copy, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&s_main2, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreateWithFlags(&join_main2, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&join_copy, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&fork, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&join_in, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&join_out, cudaEventDisableTiming) == cudaSuccess;
  const int n_out_max = kMaxChunks;
  for (int c = 0; ok && c < n_chunks; ++c)
    ok = cudaEventCreateWithFlags(&prep_done[c], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&copy_done[c], cudaEventDisableTiming) == cudaSuccess;
  for (int c = 0; ok && c < n_out_max; ++c) ok = cudaEventCreateWithFlags(&chain_done[c], cudaEventDisableTiming) == cudaSuccess;
  tq_host_stepper* hs = ok ? new tq_host_stepper() : nullptr;
  int status = ok ? TQ_OK : TQ_ERR_CUDA;
  if (ok) {
    t_capturing = true, t_captured = 0;
    const bool capturing = cudaStreamBeginCapture(s_main, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    ok = capturing && cudaEventRecord(fork, s_main) == cudaSuccess && cudaStreamWaitEvent(s_in, fork, 0) == cudaSuccess &&
         cudaStreamWaitEvent(s_out, fork, 0) == cudaSuccess && cudaStreamWaitEvent(s_copy, fork, 0) == cudaSuccess &&
         cudaStreamWaitEvent(s_main2, fork, 0) == cudaSuccess;
    // copy-in chunks grow geometrically (x 1.6): the first is short, so that the streaming chain starts after a small copy
    // and a small prep kernel, and every later chunk's copy + prep fits under the chain of the chunks in front of it.
    // The copies run on a branch of their own (a prep kernel never holds up the next copy).  Copy-out groups of
    // kOutLayers layers are independent of the chunks: a group's finish kernel and copy leave as soon as its last
    // streaming kernel is done
    int bound[kMaxChunks + 1];
    {
      double wsum = 0.0, w = 1.0, acc = 0.0;
      for (int c = 0; c < n_chunks; ++c, w *= 1.6) wsum += w;
      bound[0] = 0;
      w = 1.0;
      for (int c = 1; c <= n_chunks; ++c, w *= 1.6) {
        acc += w;
        int b = (int)(n_layers_call * acc / wsum + 0.5);
        b = b < bound[c - 1] + 1 ? bound[c - 1] + 1 : b;                                  // at least one layer per chunk
        b = b > n_layers_call - (n_chunks - c) ? n_layers_call - (n_chunks - c) : b;      // and one left for each to come
        bound[c] = c == n_chunks ? n_layers_call : b;
      }
    }
    // (a group also ends with its chunk: at most n_layers_call / out_layers + n_chunks groups, kept below kMaxChunks events)
    const int out_room = kMaxChunks - n_chunks > 1 ? kMaxChunks - n_chunks : 1;
    const int out_layers = n_layers_call > 6 * out_room ? (n_layers_call + out_room - 1) / out_room : 6;
    int out_begin = 0, n_out = 0;
    for (int c = 0; ok && c < n_chunks; ++c) {
      const int l0 = bound[c], l1 = bound[c + 1];
      const size_t off = per_layer * l0, nb = per_layer * (l1 - l0);
      if (buffers_on_host)
        ok = cudaMemcpyAsync((void*)(dk + off), (const unsigned char*)k_buf + off, nb, cudaMemcpyHostToDevice, s_copy) == cudaSuccess &&
             cudaMemcpyAsync((void*)(dv + off), (const unsigned char*)v_buf + off, nb, cudaMemcpyHostToDevice, s_copy) == cudaSuccess &&
             cudaMemcpyAsync((void*)(dq + off), (const unsigned char*)q_buf + off, nb, cudaMemcpyHostToDevice, s_copy) == cudaSuccess &&
             cudaEventRecord(copy_done[c], s_copy) == cudaSuccess && cudaStreamWaitEvent(s_in, copy_done[c], 0) == cudaSuccess;
      const DecodeArgs ca = sub_args(p, l0, l1 - l0);
      // the chains of consecutive chunks alternate between two branches: the first kernel of a chunk then waits for its prep
      // kernel only, not for the chunk in front to drain (layers are independent)
      cudaStream_t s_chain = (c & 1) ? s_main2 : s_main;
      ok = ok && launch_prep(ca, dk + off, dv + off, g.D, p.sms, true, true, s_in) == cudaSuccess &&
           cudaEventRecord(prep_done[c], s_in) == cudaSuccess && cudaStreamWaitEvent(s_chain, prep_done[c], 0) == cudaSuccess;
      for (int l = l0; ok && l < l1; ++l) {
        DecodeArgs b = sub_args(p, l, 1);
        // a captured launch with the programmatic attribute turns EVERY dependency of its stream into a programmatic
        // edge, the one to this chunk's prep kernel included (which triggers early): the first kernel of a chunk must
        // therefore wait at its start; the others run ahead
        b.chain_mode = l == l0 ? 0 : 1;
        ok = launch_decode(b, g.D, false, s_chain) == cudaSuccess;
        if (ok && (l + 1 - out_begin == out_layers || l + 1 == l1)) {  // a copy-out group is complete (groups end with the chunk)
          const DecodeArgs oa = sub_args(p, out_begin, l + 1 - out_begin);
          const size_t ooff = per_layer * out_begin, onb = per_layer * (l + 1 - out_begin);
          ok = n_out < kMaxChunks && cudaEventRecord(chain_done[n_out], s_chain) == cudaSuccess &&
               cudaStreamWaitEvent(s_out, chain_done[n_out], 0) == cudaSuccess && launch_finish(oa, g.D, false, s_out) == cudaSuccess;
          if (ok && buffers_on_host)
            ok = cudaMemcpyAsync((unsigned char*)out_buf + ooff, dout + ooff, onb, cudaMemcpyDeviceToHost, s_out) == cudaSuccess;
          out_begin = l + 1, ++n_out;
        }
      }
    }
    ok = ok && cudaEventRecord(join_main2, s_main2) == cudaSuccess && cudaStreamWaitEvent(s_main, join_main2, 0) == cudaSuccess &&
         cudaEventRecord(join_copy, s_copy) == cudaSuccess && cudaStreamWaitEvent(s_main, join_copy, 0) == cudaSuccess &&
         cudaEventRecord(join_in, s_in) == cudaSuccess && cudaStreamWaitEvent(s_main, join_in, 0) == cudaSuccess &&
         cudaEventRecord(join_out, s_out) == cudaSuccess && cudaStreamWaitEvent(s_main, join_out, 0) == cudaSuccess;
    cudaGraph_t graph = nullptr;
    if (capturing) ok = (cudaStreamEndCapture(s_main, &graph) == cudaSuccess && graph) && ok;
    if (ok) ok = cudaGraphInstantiate(&hs->exec, graph, 0) == cudaSuccess;
    hs->graph = graph;
    hs->n_launches = t_captured;  // nothing ran yet: the capture only recorded the launches
    t_capturing = false;
    if (!ok) status = TQ_ERR_CUDA;
  }
  for (int c = 0; c < kMaxChunks; ++c) {
    if (prep_done[c]) cudaEventDestroy(prep_done[c]);
    if (chain_done[c]) cudaEventDestroy(chain_done[c]);
    if (copy_done[c]) cudaEventDestroy(copy_done[c]);
  }
  if (join_copy) cudaEventDestroy(join_copy);
  if (join_main2) cudaEventDestroy(join_main2);
  if (s_copy) cudaStreamDestroy(s_copy);
  if (s_main2) cudaStreamDestroy(s_main2);
  if (fork) cudaEventDestroy(fork);
  if (join_in) cudaEventDestroy(join_in);
  if (join_out) cudaEventDestroy(join_out);
  if (s_in) cudaStreamDestroy(s_in);
  if (s_out) cudaStreamDestroy(s_out);
  if (s_main) cudaStreamDestroy(s_main);
  if (status != TQ_OK) {
    if (hs) {
      if (hs->exec) cudaGraphExecDestroy(hs->exec);
      if (hs->graph) cudaGraphDestroy(hs->graph);
      delete hs;
    }
    cudaGetLastError();
    return status;
  }
  *out_stepper = hs;
  return TQ_OK;
}

int tq_host_stepper_launch(tq_host_stepper* stepper, void* cuda_stream) {
  if (!stepper || !stepper->exec) return TQ_ERR_INVALID_ARG;
  if (cudaGraphLaunch(stepper->exec, (cudaStream_t)cuda_stream) != cudaSuccess) return TQ_ERR_CUDA;
  count_launch(stepper->n_launches);
  return TQ_OK;
}

int tq_host_stepper_run(tq_host_stepper* stepper, void* cuda_stream) {
  const int rc = tq_host_stepper_launch(stepper, cuda_stream);
  if (rc != TQ_OK) return rc;
  return cudaStreamSynchronize((cudaStream_t)cuda_stream) == cudaSuccess ? TQ_OK : TQ_ERR_CUDA;
}

int tq_host_stepper_destroy(tq_host_stepper* stepper) {
  if (!stepper) return TQ_OK;
  if (stepper->exec) cudaGraphExecDestroy(stepper->exec);
  if (stepper->graph) cudaGraphDestroy(stepper->graph);
  delete stepper;
  return TQ_OK;
}

const char* tq_status_string(int status) {
  switch (status) {
    case TQ_OK:
      return "TQ_OK";
    case TQ_ERR_INVALID_ARG:
      return "TQ_ERR_INVALID_ARG";
    case TQ_ERR_UNSUPPORTED:
      return "TQ_ERR_UNSUPPORTED";
    case TQ_ERR_CAPACITY:
      return "TQ_ERR_CAPACITY";
    case TQ_ERR_CUDA:
      return "TQ_ERR_CUDA";
    default:
      return "TQ_ERR_UNKNOWN";
  }
}

int64_t tq_launch_count(void) { return (int64_t)tq::g_launches.load(); }

#ifdef TQ_TEST_HOOKS
void tq_profile_decode_main_only(int on) { tq::g_profile_skip_prep.store(on < 0 ? 0 : (on > 2 ? 2 : on), std::memory_order_relaxed); }

void tq_debug_set_quantize_impl(int fp32_cuda_cores) { tq::debug_set_quantize_fp32(fp32_cuda_cores); }

void tq_debug_set_decode_nsplit(int nsplit) { tq::g_debug_nsplit.store(nsplit, std::memory_order_relaxed); }
#endif

}  // extern "C"
