"""ctypes front-end of the CPU ORACLE (oracle/tq_oracle.c).  TEST INFRASTRUCTURE — not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It marshals numpy arrays into the plain-C oracle and back; it holds no arithmetic of the method
(the two calibration helpers call numpy's SVD / QR as library primitives, as PAPER.md:132-137 and
BASELINE.json:configs[0] define the rotation).  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tq_oracle.c")
_LIB = os.path.join(_HERE, "libtqo.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/tq_oracle.c with gcc (-O2, OpenMP over independent units)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.tqo_f16_to_f64.restype = C.c_double
        _lib.tqo_f16_to_f64.argtypes = [C.c_uint16]
        _lib.tqo_f64_to_f16.restype = C.c_uint16
        _lib.tqo_f64_to_f16.argtypes = [C.c_double]
        _lib.tqo_qjl_estimate.restype = C.c_double
        _lib.tqo_lloyd_max_gauss.restype = C.c_double
        _lib.tqo_lloyd_max_samples.restype = C.c_double
        _lib.tqo_code.restype = C.c_int
        _lib.tqo_code_argmin.restype = C.c_int
        _lib.tqo_num_threads.restype = C.c_int
    return _lib


def _p(a, ty=None):
    if a is None:
        return None
    assert a.flags["C_CONTIGUOUS"], "oracle arrays must be C-contiguous"
    return a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().tqo_num_threads())


def set_num_threads(n: int) -> None:
    lib().tqo_set_num_threads(C.c_int(int(n)))


# ---------------------------------------------------------------------------------------------------
# scalar helpers
def f64_to_f16_bits(x: float) -> int:
    return int(lib().tqo_f64_to_f16(C.c_double(float(x))))


def f16_bits_to_f64(h: int) -> float:
    return float(lib().tqo_f16_to_f64(C.c_uint16(int(h))))


def rope(x, pos: float, base: float = 10000.0, layout: int = 0):
    x = _f64(x)
    out = np.empty_like(x)
    lib().tqo_rope(_p(x), C.c_int(x.shape[-1]), C.c_double(pos), C.c_double(base), C.c_int(layout), _p(out))
    return out


def code(u: float, lut8) -> int:
    lut8 = _f32(lut8)
    return int(lib().tqo_code(C.c_double(float(u)), _p(lut8)))


def code_argmin(u: float, lut8) -> int:
    lut8 = _f32(lut8)
    return int(lib().tqo_code_argmin(C.c_double(float(u)), _p(lut8)))


def pack_codes(codes):
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    d = codes.shape[-1]
    out = np.empty(3 * d // 8, dtype=np.uint8)
    lib().tqo_pack_codes(_p(codes), C.c_int(d), _p(out))
    return out


def unpack_codes(packed, d: int):
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    out = np.empty(d, dtype=np.uint8)
    lib().tqo_unpack_codes(_p(packed), C.c_int(d), _p(out))
    return out


def pack_bits(bits):
    bits = np.ascontiguousarray(bits, dtype=np.uint8)
    m = bits.shape[-1]
    out = np.empty(m // 8, dtype=np.uint8)
    lib().tqo_pack_bits(_p(bits), C.c_int(m), _p(out))
    return out


def unpack_bits(packed, m: int):
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    out = np.empty(m, dtype=np.uint8)
    lib().tqo_unpack_bits(_p(packed), C.c_int(m), _p(out))
    return out


def quantize_vector(x, is_key: bool, pos: float, Pi, lut8, S, base: float = 10000.0, layout: int = 0):
    """One vector -> dict(codes[d], bits[m], norm_h, rnorm_h, u[d])."""
    x = _f64(x)
    d = x.shape[0]
    S = _f32(S)
    m = S.shape[0]
    Pi = _f32(Pi)
    lut8 = _f32(lut8)
    codes = np.zeros(d, np.uint8)
    bits = np.zeros(m, np.uint8)
    nh = C.c_uint16(0)
    rh = C.c_uint16(0)
    u = np.zeros(d, np.float64)
    lib().tqo_quantize_vector(_p(x), C.c_int(d), C.c_int(m), C.c_int(1 if is_key else 0), C.c_double(pos),
                              C.c_double(base), C.c_int(layout), _p(Pi), _p(lut8), _p(S), _p(codes), _p(bits),
                              C.byref(nh), C.byref(rh), _p(u))
    return dict(codes=codes, bits=bits, norm_h=nh.value, rnorm_h=rh.value, u=u)


def key_sketch_values(kvec, pos, Pi, lut8, S, base=10000.0, layout=0):
    kvec = _f32(kvec)
    S = _f32(S)
    m, d = S.shape
    out = np.zeros(m, np.float64)
    Pi = _f32(Pi)
    lut8 = _f32(lut8)
    lib().tqo_key_sketch_values(_p(kvec), C.c_int(d), C.c_int(m), C.c_double(pos), C.c_double(base),
                                C.c_int(layout), _p(Pi), _p(lut8), _p(S), _p(out))
    return out


def qjl_estimate(q, r, S) -> float:
    q = _f64(q)
    r = _f64(r)
    S = _f32(S)
    m, d = S.shape
    return float(lib().tqo_qjl_estimate(_p(q), _p(r), _p(S), C.c_int(m), C.c_int(d)))


def dequant_vector(packed_codes, norm_h: int, Pi, lut8, unrotate: bool = True):
    packed_codes = np.ascontiguousarray(packed_codes, dtype=np.uint8)
    Pi = _f32(Pi)
    d = Pi.shape[0]
    lut8 = _f32(lut8)
    out = np.zeros(d, np.float64)
    lib().tqo_dequant_vector(_p(packed_codes), C.c_uint16(int(norm_h)), C.c_int(d), _p(Pi), _p(lut8),
                             C.c_int(1 if unrotate else 0), _p(out))
    return out


# ---------------------------------------------------------------------------------------------------
# calibration pieces
def lloyd_max_gauss(sigma: float, levels: int = 8, iters: int = 500):
    """Fixed point of Eq. 5 for N(0, sigma^2) -> (centroids, thresholds, mse/sigma^2)."""
    c = np.zeros(levels, np.float64)
    t = np.zeros(levels - 1, np.float64)
    mse = lib().tqo_lloyd_max_gauss(C.c_double(sigma), C.c_int(levels), C.c_int(iters), _p(c), _p(t))
    return c, t, float(mse)


def lloyd_max_samples(samples, levels: int = 8, iters: int = 100):
    s = np.sort(_f64(samples).ravel())
    c = np.zeros(levels, np.float64)
    mse = lib().tqo_lloyd_max_samples(_p(s), C.c_long(s.shape[0]), C.c_int(levels), C.c_int(iters), _p(c))
    return c, float(mse)


def svd_rotation(X):
    """X = U Sigma V^T (uncentred, N_cal x d) -> PI = V^T.  numpy's SVD is the library
    primitive; singular-vector signs are not unique (D9)."""
    _, _, vt = np.linalg.svd(_f64(X), full_matrices=False)
    return vt


# ---------------------------------------------------------------------------------------------------
# whole-layer calls
@dataclass
class Canonical:
    """Canonical packed planes of one layer, index [b][h][t] (include/tq.h 'Canonical packed format')."""
    k_codes: np.ndarray  # [B,H,T,3d/8] u8
    k_signs: np.ndarray  # [B,H,T,m/8]  u8
    k_norm: np.ndarray   # [B,H,T] u16
    k_rnorm: np.ndarray  # [B,H,T] u16
    v_codes: np.ndarray  # [B,H,T,3d/8] u8
    v_norm: np.ndarray   # [B,H,T] u16
    near_k: np.ndarray | None = None  # [B,H,T,d] u8
    near_v: np.ndarray | None = None
    v_signs: np.ndarray | None = None  # [B,H,T,m/8] u8   (V-side sketch, tq_shape.v_qjl = 1)
    v_rnorm: np.ndarray | None = None  # [B,H,T] u16


def quantize_pack(k, v, pi_k, pi_v, lut_k, lut_v, S, start_pos: int = 0, base: float = 10000.0,
                  layout: int = 0, near_eps: float | None = None) -> Canonical:
    """k, v: [B,H,T,d] (fp16 or fp32, widened exactly); pi_*: [H,d,d]; lut_*: [H,8]; S: [m,d]."""
    k = _f32(k)
    v = _f32(v)
    B, H, T, d = k.shape
    S = _f32(S)
    m = S.shape[0]
    pi_k, pi_v, lut_k, lut_v = _f32(pi_k), _f32(pi_v), _f32(lut_k), _f32(lut_v)
    assert pi_k.shape == (H, d, d) and lut_k.shape == (H, 8)
    cb, sb = 3 * d // 8, m // 8
    out = Canonical(np.zeros((B, H, T, cb), np.uint8), np.zeros((B, H, T, sb), np.uint8),
                    np.zeros((B, H, T), np.uint16), np.zeros((B, H, T), np.uint16),
                    np.zeros((B, H, T, cb), np.uint8), np.zeros((B, H, T), np.uint16))
    if near_eps is not None:
        out.near_k = np.zeros((B, H, T, d), np.uint8)
        out.near_v = np.zeros((B, H, T, d), np.uint8)
    lib().tqo_quantize_pack(C.c_int(B), C.c_int(H), C.c_int(T), C.c_int(d), C.c_int(m), C.c_double(base),
                            C.c_int(layout), C.c_int(start_pos), _p(k), _p(v), _p(pi_k), _p(pi_v), _p(lut_k),
                            _p(lut_v), _p(S), _p(out.k_codes), _p(out.k_signs), _p(out.k_norm), _p(out.k_rnorm),
                            _p(out.v_codes), _p(out.v_norm), C.c_double(near_eps or 0.0), _p(out.near_k),
                            _p(out.near_v))
    return out


def quantize_vector_literal(x, is_key: bool, pos: float, Pi, lut8, S, ebar: float, base: float = 10000.0, layout: int = 0):
    """Paper-literal Eq. 6-7 mode, one vector -> dict(codes[d], bits[m], norm_h, rnorm_h, y[d])."""
    x = _f64(x)
    d = x.shape[0]
    S = _f32(S)
    m = S.shape[0]
    codes, bits = np.zeros(d, np.uint8), np.zeros(m, np.uint8)
    nh, rh = C.c_uint16(0), C.c_uint16(0)
    y = np.zeros(d, np.float64)
    lib().tqo_quantize_vector_literal(_p(x), C.c_int(d), C.c_int(m), C.c_int(1 if is_key else 0), C.c_double(pos),
                                      C.c_double(base), C.c_int(layout), _p(_f32(Pi)), _p(_f32(lut8)), _p(S),
                                      C.c_double(ebar), _p(codes), _p(bits), C.byref(nh), C.byref(rh), _p(y))
    return dict(codes=codes, bits=bits, norm_h=nh.value, rnorm_h=rh.value, y=y)


def quantize_pack_literal(k, v, pi_k, pi_v, lut_k, lut_v, S, ebar_k, start_pos: int = 0, base: float = 10000.0,
                          layout: int = 0, near_eps: float | None = None) -> Canonical:
    """Layer form of the paper-literal mode; ebar_k: [H].  Same planes as quantize_pack."""
    k = _f32(k)
    v = _f32(v)
    B, H, T, d = k.shape
    S = _f32(S)
    m = S.shape[0]
    pi_k, pi_v, lut_k, lut_v, ebar_k = _f32(pi_k), _f32(pi_v), _f32(lut_k), _f32(lut_v), _f32(ebar_k)
    assert pi_k.shape == (H, d, d) and lut_k.shape == (H, 8) and ebar_k.shape == (H,)
    cb, sb = 3 * d // 8, m // 8
    out = Canonical(np.zeros((B, H, T, cb), np.uint8), np.zeros((B, H, T, sb), np.uint8),
                    np.zeros((B, H, T), np.uint16), np.zeros((B, H, T), np.uint16),
                    np.zeros((B, H, T, cb), np.uint8), np.zeros((B, H, T), np.uint16))
    if near_eps is not None:
        out.near_k = np.zeros((B, H, T, d), np.uint8)
        out.near_v = np.zeros((B, H, T, d), np.uint8)
    lib().tqo_quantize_pack_literal(C.c_int(B), C.c_int(H), C.c_int(T), C.c_int(d), C.c_int(m), C.c_double(base),
                                    C.c_int(layout), C.c_int(start_pos), _p(k), _p(v), _p(pi_k), _p(pi_v), _p(lut_k),
                                    _p(lut_v), _p(S), _p(ebar_k), _p(out.k_codes), _p(out.k_signs), _p(out.k_norm),
                                    _p(out.k_rnorm), _p(out.v_codes), _p(out.v_norm), C.c_double(near_eps or 0.0),
                                    _p(out.near_k), _p(out.near_v))
    return out


def add_value_sketch(can: Canonical, v, pi_v, lut_v, S) -> Canonical:
    """V-side residual sketch planes (Algorithm 1 line 10): fills can.v_signs / can.v_rnorm."""
    v = _f32(v)
    B, H, T, d = v.shape
    S = _f32(S)
    m = S.shape[0]
    can.v_signs = np.zeros((B, H, T, m // 8), np.uint8)
    can.v_rnorm = np.zeros((B, H, T), np.uint16)
    lib().tqo_value_sketch_planes(C.c_int(B), C.c_int(H), C.c_int(T), C.c_int(d), C.c_int(m), _p(v), _p(_f32(pi_v)),
                                  _p(_f32(lut_v)), _p(S), _p(can.v_signs), _p(can.v_rnorm))
    return can


def decode_attn_vq(q, q_pos, seq_len, pi_k, pi_v, lut_k, lut_v, S, cache: Canonical, base: float = 10000.0,
                   layout: int = 0):
    """decode_attn with the V-side sketch: values are n (lut_V[codes] + sqrt(pi/2)/m |r| S^T sigma)."""
    q = _f32(q)
    B, H, d = q.shape
    S = _f32(S)
    m = S.shape[0]
    T_stride = cache.k_norm.shape[2]
    q_pos = np.ascontiguousarray(q_pos, dtype=np.int32)
    seq_len = np.ascontiguousarray(seq_len, dtype=np.int32)
    assert int(seq_len.max(initial=0)) <= T_stride and cache.v_signs is not None
    out = np.zeros((B, H, d), np.float64)
    c = np.ascontiguousarray
    lib().tqo_decode_attn_vq(C.c_int(B), C.c_int(H), C.c_int(d), C.c_int(m), C.c_int(T_stride), C.c_double(base),
                             C.c_int(layout), _p(q), _p(q_pos), _p(seq_len), _p(_f32(pi_k)), _p(_f32(pi_v)), _p(_f32(lut_k)),
                             _p(_f32(lut_v)), _p(S), _p(c(cache.k_codes)), _p(c(cache.k_signs)), _p(c(cache.k_norm)),
                             _p(c(cache.k_rnorm)), _p(c(cache.v_codes)), _p(c(cache.v_norm)), _p(c(cache.v_signs)),
                             _p(c(cache.v_rnorm)), _p(out))
    return out


def decode_attn(q, q_pos, seq_len, pi_k, pi_v, lut_k, lut_v, S, cache: Canonical, base: float = 10000.0,
                layout: int = 0, use_qjl: bool = True):
    """q: [B,H,d]; q_pos, seq_len: [B] int32 -> out [B,H,d] fp64."""
    q = _f32(q)
    B, H, d = q.shape
    S = _f32(S)
    m = S.shape[0]
    T_stride = cache.k_norm.shape[2]
    q_pos = np.ascontiguousarray(q_pos, dtype=np.int32)
    seq_len = np.ascontiguousarray(seq_len, dtype=np.int32)
    assert int(seq_len.max(initial=0)) <= T_stride
    pi_k, pi_v, lut_k, lut_v = _f32(pi_k), _f32(pi_v), _f32(lut_k), _f32(lut_v)
    out = np.zeros((B, H, d), np.float64)
    lib().tqo_decode_attn(C.c_int(B), C.c_int(H), C.c_int(d), C.c_int(m), C.c_int(T_stride), C.c_double(base),
                          C.c_int(layout), _p(q), _p(q_pos), _p(seq_len), _p(pi_k), _p(pi_v), _p(lut_k),
                          _p(lut_v), _p(S), _p(np.ascontiguousarray(cache.k_codes)),
                          _p(np.ascontiguousarray(cache.k_signs)), _p(np.ascontiguousarray(cache.k_norm)),
                          _p(np.ascontiguousarray(cache.k_rnorm)), _p(np.ascontiguousarray(cache.v_codes)),
                          _p(np.ascontiguousarray(cache.v_norm)), C.c_int(1 if use_qjl else 0), _p(out))
    return out


def dense_attn_ref(q, q_pos, seq_len, k, v, base: float = 10000.0, layout: int = 0):
    """Exact fp64 attention on the original tensors (Eq. 1): q [B,H,d], k/v [B,H,T,d] -> [B,H,d]."""
    q = _f32(q)
    k = _f32(k)
    v = _f32(v)
    B, H, d = q.shape
    T_stride = k.shape[2]
    q_pos = np.ascontiguousarray(q_pos, dtype=np.int32)
    seq_len = np.ascontiguousarray(seq_len, dtype=np.int32)
    out = np.zeros((B, H, d), np.float64)
    lib().tqo_dense_attn_ref(C.c_int(B), C.c_int(H), C.c_int(d), C.c_int(T_stride), C.c_double(base),
                             C.c_int(layout), _p(q), _p(q_pos), _p(seq_len), _p(k), _p(v), _p(out))
    return out
