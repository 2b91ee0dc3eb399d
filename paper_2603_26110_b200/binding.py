"""Thin ctypes binding of libtq.so (include/tq.h).  Argument marshalling only: every step of the hot path
runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams, nothing else.

There is no CPU fallback: if libtq.so is missing this module raises at first use, and every device entry
point returns TQ_ERR_CUDA (raised here as TqError) when no CUDA device is usable.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtq.so")

TQ_OK, TQ_ERR_INVALID_ARG, TQ_ERR_UNSUPPORTED, TQ_ERR_CAPACITY, TQ_ERR_CUDA = 0, 1, 2, 3, 4
TQ_F16, TQ_F32 = 0, 1
TILE_TOKENS = 32

EXPORTS = [
    "tq_cache_bytes", "tq_cache_bytes_per_token_head", "tq_cache_seq_len_offset", "tq_cache_status_offset",
    "tq_decode_workspace_bytes", "tq_canonical_plane_bytes", "tq_calibrate_host", "tq_quantize_pack", "tq_append",
    "tq_decode_attn", "tq_decode_attn_noalloc", "tq_noalloc_scratch_bytes", "tq_decode_step", "tq_cache_export_canonical", "tq_cache_import_canonical", "tq_step_staging_bytes",
    "tq_decode_step_host", "tq_model_step_staging_bytes", "tq_decode_model_step_host", "tq_decode_model_step", "tq_status_string", "tq_launch_count", "tq_profile_decode_main_only",
    "tq_debug_set_decode_nsplit", "tq_debug_set_quantize_impl", "tq_host_stepper_create", "tq_host_stepper_launch", "tq_host_stepper_run",
    "tq_host_stepper_destroy",
]


class TqError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)}")


class TqShape(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("batch", C.c_int32), ("n_heads", C.c_int32), ("head_dim", C.c_int32),
                ("qjl_dim", C.c_int32), ("max_seq", C.c_int32), ("rope_base", C.c_float), ("rope_layout", C.c_int32),
                ("v_qjl", C.c_int32), ("residual_mode", C.c_int32)]


class TqParams(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("pi_k", "pi_v", "lut_k", "lut_v", "S", "rope_cs", "ebar_k")]


class TqCache(C.Structure):
    _fields_ = [("data", C.c_void_p)]


class TqCanonical(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("k_codes", "k_signs", "k_norm", "k_rnorm", "v_codes", "v_norm", "v_signs", "v_rnorm")]


_lib = None


def lib():
    """Load libtq.so; fail loudly when the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build the CUDA extension first (python -m paper_2603_26110_b200.build). "
                "There is no CPU fallback.")
        l = C.CDLL(LIB_PATH)
        for n in ("tq_cache_bytes", "tq_cache_bytes_per_token_head", "tq_cache_seq_len_offset",
                  "tq_cache_status_offset", "tq_decode_workspace_bytes", "tq_canonical_plane_bytes",
                  "tq_step_staging_bytes", "tq_model_step_staging_bytes", "tq_noalloc_scratch_bytes"):
            getattr(l, n).restype = C.c_size_t
        l.tq_status_string.restype = C.c_char_p
        l.tq_launch_count.restype = C.c_int64
        _lib = l
    return _lib


def status_string(status: int) -> str:
    return lib().tq_status_string(C.c_int(status)).decode()


def _check(rc: int, where: str):
    if rc != TQ_OK:
        raise TqError(rc, where)


def make_shape(n_layers, batch, n_heads, head_dim, max_seq, rope_base=10000.0, rope_layout=0, qjl_dim=None,
               v_qjl=0, residual_mode=0) -> TqShape:
    return TqShape(n_layers, batch, n_heads, head_dim, head_dim if qjl_dim is None else qjl_dim, max_seq, rope_base,
                   rope_layout, v_qjl, residual_mode)


def _ptr(t):
    """data pointer of a torch tensor / numpy array / None"""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _dtype_code(t) -> int:
    import torch

    if t.dtype == torch.float16:
        return TQ_F16
    if t.dtype == torch.float32:
        return TQ_F32
    raise TypeError(f"q/k/v must be float16 or float32, got {t.dtype}")


def _stream_ptr(stream=None):
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


# ---- sizes --------------------------------------------------------------------------------------------
def tq_cache_bytes(shape: TqShape) -> int:
    return int(lib().tq_cache_bytes(C.byref(shape)))


def tq_cache_bytes_per_token_head(shape: TqShape) -> int:
    return int(lib().tq_cache_bytes_per_token_head(C.byref(shape)))


def tq_decode_workspace_bytes(shape: TqShape, n_layers_call: int) -> int:
    return int(lib().tq_decode_workspace_bytes(C.byref(shape), C.c_int32(n_layers_call)))


def tq_canonical_plane_bytes(shape: TqShape, plane: int, n_tokens: int) -> int:
    return int(lib().tq_canonical_plane_bytes(C.byref(shape), C.c_int32(plane), C.c_int32(n_tokens)))


def tq_step_staging_bytes(shape: TqShape, dt: int) -> int:
    return int(lib().tq_step_staging_bytes(C.byref(shape), C.c_int(dt)))


def tq_launch_count() -> int:
    return int(lib().tq_launch_count())


def tq_profile_decode_main_only(on: bool):
    """Measurement hook: tq_decode_attn launches only the streaming kernel (queries from the previous ordinary call)."""
    lib().tq_profile_decode_main_only(C.c_int(int(on)))  # 0 off, 1 skip the prep kernel, 2 also skip the finish kernel


# ---- calibration (host) -------------------------------------------------------------------------------
def tq_calibrate_host(shape: TqShape, mode: int, k_samples=None, v_samples=None, seed: int = 0) -> dict:
    """Returns host numpy arrays pi_k, pi_v [L,H,d,d], lut_k, lut_v [L,H,8], S [m,d], rope_cs [max_seq,d/2,2]."""
    L, H, d, m = shape.n_layers, shape.n_heads, shape.head_dim, shape.qjl_dim
    out = dict(pi_k=np.zeros((L, H, d, d), np.float32), pi_v=np.zeros((L, H, d, d), np.float32),
               lut_k=np.zeros((L, H, 8), np.float32), lut_v=np.zeros((L, H, 8), np.float32),
               S=np.zeros((m, d), np.float32), rope_cs=np.zeros((shape.max_seq, d // 2, 2), np.float32))
    if shape.residual_mode == 1:
        out["ebar_k"] = np.zeros((L, H), np.float32)
    p = TqParams(*[C.c_void_p(out[n].ctypes.data) if n in out else None
                   for n in ("pi_k", "pi_v", "lut_k", "lut_v", "S", "rope_cs", "ebar_k")])
    n_samples = 0
    if k_samples is not None:
        k_samples = np.ascontiguousarray(k_samples, np.float32)
        v_samples = np.ascontiguousarray(v_samples, np.float32)
        n_samples = k_samples.shape[2]
    rc = lib().tq_calibrate_host(C.byref(shape), C.c_int32(mode), _ptr(k_samples), _ptr(v_samples),
                                 C.c_int64(n_samples), C.c_uint64(seed), C.byref(p))
    _check(rc, "tq_calibrate_host")
    return out


# ---- device-side holders (plumbing: torch owns the memory) ----------------------------------------------
class Params:
    """Calibration arrays resident on the device + the C struct that points at them."""

    def __init__(self, arrays: dict, device="cuda"):
        import torch

        names = ("pi_k", "pi_v", "lut_k", "lut_v", "S", "rope_cs", "ebar_k")  # ebar_k: paper-literal mode only
        self.t = {n: torch.as_tensor(np.ascontiguousarray(arrays[n], np.float32)).to(device).contiguous()
                  for n in names if arrays.get(n) is not None}
        self.c = TqParams(*[C.c_void_p(self.t[n].data_ptr()) if n in self.t else None for n in names])


class Cache:
    """One zero-filled device buffer of tq_cache_bytes(shape) bytes."""

    def __init__(self, shape: TqShape, device="cuda"):
        import torch

        self.shape = shape
        n = tq_cache_bytes(shape)
        if n == 0:
            raise TqError(TQ_ERR_INVALID_ARG, "tq_cache_bytes")
        self.buf = torch.zeros(n + 256, dtype=torch.uint8, device=device)
        off = (-self.buf.data_ptr()) % 256
        self.data = self.buf[off:off + n]
        self.c = TqCache(C.c_void_p(self.data.data_ptr()))
        so = int(lib().tq_cache_seq_len_offset(C.byref(shape)))
        self.seq_len = self.data[so:so + 4 * shape.n_layers * shape.batch].view(torch.int32).view(shape.n_layers, shape.batch)
        st = int(lib().tq_cache_status_offset(C.byref(shape)))
        self.status = self.data[st:st + 4].view(torch.int32)


class Workspace:
    def __init__(self, shape: TqShape, n_layers_call: int, device="cuda"):
        import torch

        self.bytes = tq_decode_workspace_bytes(shape, n_layers_call)
        if self.bytes == 0:
            raise TqError(TQ_ERR_INVALID_ARG, "tq_decode_workspace_bytes")
        self.buf = torch.zeros(self.bytes + 256, dtype=torch.uint8, device=device)
        off = (-self.buf.data_ptr()) % 256
        self.data = self.buf[off:off + self.bytes]


# ---- hot-path calls --------------------------------------------------------------------------------------
def tq_quantize_pack(shape, params: Params, cache: Cache, layer: int, k, v, start_pos: int = 0, stream=None):
    """k, v: device tensors [B,H,T,d] (fp16 or fp32)."""
    n_tokens = int(k.shape[2])
    rc = lib().tq_quantize_pack(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer), _ptr(k), _ptr(v),
                                C.c_int(_dtype_code(k)), C.c_int32(n_tokens), C.c_int32(start_pos), _stream_ptr(stream))
    _check(rc, "tq_quantize_pack")


def tq_append(shape, params: Params, cache: Cache, layer: int, k, v, stream=None):
    """k, v: device tensors [B,H,d]."""
    rc = lib().tq_append(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer), _ptr(k), _ptr(v),
                         C.c_int(_dtype_code(k)), _stream_ptr(stream))
    _check(rc, "tq_append")


def tq_decode_attn(shape, params: Params, cache: Cache, layer_begin: int, n_layers_call: int, q, out, workspace: Workspace,
                   q_pos=None, t_hint: int = 0, stream=None):
    """q, out: device tensors [Lc,B,H,d]; q_pos: device int32 [Lc,B] or None."""
    rc = lib().tq_decode_attn(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer_begin),
                              C.c_int32(n_layers_call), _ptr(q), _ptr(q_pos), C.c_int(_dtype_code(q)), _ptr(out),
                              C.c_int32(t_hint), _ptr(workspace.data), C.c_size_t(workspace.bytes), _stream_ptr(stream))
    _check(rc, "tq_decode_attn")


def tq_noalloc_scratch_bytes() -> int:
    """Size of the workspace array built into the library (the limit of tq_decode_attn_noalloc)."""
    return int(lib().tq_noalloc_scratch_bytes())


def tq_decode_attn_noalloc(shape, params: Params, cache: Cache, layer_begin: int, n_layers_call: int, q, out, q_pos=None,
                           t_hint: int = 0, stream=None):
    """tq_decode_attn for a caller that has no way of allocating the workspace (a plug-in inside an application whose
    memory pool owns the device, code on a path where cudaMalloc's device-wide synchronisation is not allowed, a process
    whose HBM is already given away): the workspace is a 24 MiB array built into libtq.so, so there is no `workspace`
    argument and the call allocates nothing.  q, out, q_pos as in tq_decode_attn.  A shape whose workspace exceeds
    tq_noalloc_scratch_bytes() is refused (TqError, TQ_ERR_CAPACITY) before anything is launched.  All such calls on one
    device share the array: keep them on one stream (overlapping calls race).  The first call on a device looks up the
    array's address; make it before any stream capture."""
    need = tq_decode_workspace_bytes(shape, n_layers_call)
    rc = lib().tq_decode_attn_noalloc(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer_begin),
                                      C.c_int32(n_layers_call), _ptr(q), _ptr(q_pos), C.c_int(_dtype_code(q)), _ptr(out),
                                      C.c_int32(t_hint), _stream_ptr(stream))
    if rc == TQ_ERR_CAPACITY:
        raise TqError(rc, f"tq_decode_attn_noalloc: this shape needs {need} bytes of workspace, the array built into "
                          f"the library holds {tq_noalloc_scratch_bytes()} (use fewer layers per call, or tq_decode_attn "
                          "with a workspace of your own)")
    _check(rc, "tq_decode_attn_noalloc")


def tq_decode_step(shape, params: Params, cache: Cache, layer: int, q, k, v, out, workspace: Workspace, t_hint: int = 0,
                   stream=None):
    """q, k, v, out: device tensors [B,H,d]: append (k, v), then attend with q at the new position."""
    rc = lib().tq_decode_step(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer), _ptr(q), _ptr(k),
                              _ptr(v), C.c_int(_dtype_code(q)), _ptr(out), C.c_int32(t_hint), _ptr(workspace.data),
                              C.c_size_t(workspace.bytes), _stream_ptr(stream))
    _check(rc, "tq_decode_step")


def tq_decode_model_step(shape, params: Params, cache: Cache, layer_begin: int, n_layers_call: int, q, k, v, out,
                         workspace: Workspace, t_hint: int = 0, stream=None):
    """q, k, v, out: device tensors [Lc,B,H,d]: one decode step of Lc consecutive layers (workspace for Lc layers)."""
    rc = lib().tq_decode_model_step(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer_begin),
                                    C.c_int32(n_layers_call), _ptr(q), _ptr(k), _ptr(v), C.c_int(_dtype_code(q)), _ptr(out),
                                    C.c_int32(t_hint), _ptr(workspace.data), C.c_size_t(workspace.bytes), _stream_ptr(stream))
    _check(rc, "tq_decode_model_step")


def tq_debug_set_decode_nsplit(nsplit: int):
    """Test / sweep knob: CTAs per unit of the streaming decode kernel (0 = the library's own plan)."""
    lib().tq_debug_set_decode_nsplit(C.c_int(nsplit))


def tq_debug_set_quantize_impl(fp32_cuda_cores: bool):
    """Test knob: route tq_quantize_pack to the fp32 CUDA-core kernel (cross-check of the tensor-core kernel)."""
    lib().tq_debug_set_quantize_impl(C.c_int(int(fp32_cuda_cores)))


def _canon_struct(planes: dict) -> TqCanonical:
    return TqCanonical(*[_ptr(planes.get(n)) for n in ("k_codes", "k_signs", "k_norm", "k_rnorm", "v_codes", "v_norm",
                                                       "v_signs", "v_rnorm")])


def alloc_canonical(shape, n_tokens: int, device="cuda") -> dict:
    import torch

    B, H, d, m = shape.batch, shape.n_heads, shape.head_dim, shape.qjl_dim
    extra = {}
    if shape.v_qjl == 1:  # V-side sketch planes
        extra = dict(v_signs=torch.zeros((B, H, n_tokens, m // 8), dtype=torch.uint8, device=device),
                     v_rnorm=torch.zeros((B, H, n_tokens), dtype=torch.int16, device=device))
    return dict(**extra, k_codes=torch.zeros((B, H, n_tokens, 3 * d // 8), dtype=torch.uint8, device=device),
                k_signs=torch.zeros((B, H, n_tokens, m // 8), dtype=torch.uint8, device=device),
                k_norm=torch.zeros((B, H, n_tokens), dtype=torch.int16, device=device),
                k_rnorm=torch.zeros((B, H, n_tokens), dtype=torch.int16, device=device),
                v_codes=torch.zeros((B, H, n_tokens, 3 * d // 8), dtype=torch.uint8, device=device),
                v_norm=torch.zeros((B, H, n_tokens), dtype=torch.int16, device=device))


def tq_cache_export_canonical(shape, cache: Cache, layer: int, n_tokens: int, planes: dict | None = None, stream=None) -> dict:
    planes = alloc_canonical(shape, n_tokens, cache.data.device) if planes is None else planes
    cs = _canon_struct(planes)
    rc = lib().tq_cache_export_canonical(C.byref(shape), C.byref(cache.c), C.c_int32(layer), C.c_int32(n_tokens),
                                         C.byref(cs), _stream_ptr(stream))
    _check(rc, "tq_cache_export_canonical")
    return planes


def tq_cache_import_canonical(shape, cache: Cache, layer: int, n_tokens: int, planes: dict, stream=None):
    cs = _canon_struct(planes)
    rc = lib().tq_cache_import_canonical(C.byref(shape), C.byref(cache.c), C.c_int32(layer), C.c_int32(n_tokens),
                                         C.byref(cs), _stream_ptr(stream))
    _check(rc, "tq_cache_import_canonical")


def tq_decode_step_host(shape, params: Params, cache: Cache, layer: int, q_host, k_host, v_host, out_host, staging,
                        workspace: Workspace, t_hint: int = 0, stream=None):
    """Host (pinned) tensors q/k/v/out [B,H,d]; copies + tq_append + tq_decode_attn + copy back + stream sync."""
    rc = lib().tq_decode_step_host(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer), _ptr(q_host),
                                   _ptr(k_host), _ptr(v_host), C.c_int(_dtype_code(q_host)), _ptr(out_host),
                                   C.c_int32(t_hint), _ptr(staging), _ptr(workspace.data), C.c_size_t(workspace.bytes),
                                   _stream_ptr(stream))
    _check(rc, "tq_decode_step_host")


def tq_model_step_staging_bytes(shape: TqShape, dt: int, n_layers_call: int) -> int:
    return int(lib().tq_model_step_staging_bytes(C.byref(shape), C.c_int(dt), C.c_int32(n_layers_call)))


def tq_decode_model_step_host(shape, params: Params, cache: Cache, layer_begin: int, n_layers_call: int, q_host, k_host,
                              v_host, out_host, staging, workspace: Workspace, t_hint: int = 0, stream=None):
    """Host (pinned) tensors q/k/v/out [Lc,B,H,d]: three copies in, a decode step per layer, one copy out, one sync."""
    rc = lib().tq_decode_model_step_host(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer_begin),
                                         C.c_int32(n_layers_call), _ptr(q_host), _ptr(k_host), _ptr(v_host),
                                         C.c_int(_dtype_code(q_host)), _ptr(out_host), C.c_int32(t_hint), _ptr(staging),
                                         _ptr(workspace.data), C.c_size_t(workspace.bytes), _stream_ptr(stream))
    _check(rc, "tq_decode_model_step_host")


class HostStepper:
    """tq_host_stepper_*: the model decode step captured once as a CUDA graph (copy-in / streaming chain / copy-out
    branches).  q/k/v/out: pinned HOST tensors [Lc,B,H,d] (copies recorded; staging required) or DEVICE tensors (no
    copies); the caller re-fills q/k/v before every run()."""

    def __init__(self, shape, params: Params, cache: Cache, layer_begin: int, n_layers_call: int, q, k, v, out, staging,
                 workspace: Workspace, t_hint: int = 0, n_chunks: int = 0):
        self._keep = (shape, params, cache, q, k, v, out, staging, workspace)
        on_host = 0 if q.is_cuda else 1
        self.h = C.c_void_p()
        rc = lib().tq_host_stepper_create(C.byref(shape), C.byref(params.c), C.byref(cache.c), C.c_int32(layer_begin),
                                          C.c_int32(n_layers_call), _ptr(q), _ptr(k), _ptr(v), _ptr(out), C.c_int32(on_host),
                                          C.c_int(_dtype_code(q)), C.c_int32(t_hint), _ptr(staging), _ptr(workspace.data),
                                          C.c_size_t(workspace.bytes), C.c_int32(n_chunks), C.byref(self.h))
        _check(rc, "tq_host_stepper_create")

    def launch(self, stream=None):
        """asynchronous: one graph launch"""
        _check(lib().tq_host_stepper_launch(self.h, _stream_ptr(stream)), "tq_host_stepper_launch")

    def run(self, stream=None):
        """graph launch + stream synchronisation"""
        _check(lib().tq_host_stepper_run(self.h, _stream_ptr(stream)), "tq_host_stepper_run")

    def close(self):
        if self.h:
            lib().tq_host_stepper_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
