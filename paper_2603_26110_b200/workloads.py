"""Seeded synthetic workloads shaped like BASELINE.json:configs[0..4].

This module serves BOTH the CPU oracle's tests and the CUDA path, so it holds none of the method's
arithmetic: it only draws random numbers (numpy Generator(PCG64)) and shapes them.  The rotation matrices
are the Q factors of seeded Gaussian matrices as configs[0]/[1] prescribe (numpy's QR is the library
primitive); LUTs are NOT produced here — callers pass them in as data (tests take them from the oracle's
Lloyd-Max, the product from tq_calibrate_host).

The inputs stand in for ESM-2 activations on real proteins, which are not available:
heavy-tailed Student-t(4) or Gaussian coordinates with a few fixed per-head outlier channels
("channel-wise outliers").
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

SEED0 = 260326110


@dataclass(frozen=True)
class Workload:
    name: str
    index: int          # BASELINE.json configs[index]
    n_layers: int
    batch: int
    n_heads: int
    head_dim: int
    seq: int            # cached tokens per (layer, batch, head)
    dtype: str          # "f32" | "f16"
    dist: str           # "normal" | "student_t4"
    n_outlier: int      # outlier channels per head
    outlier_scale: float
    fixed_outliers: tuple = ()   # explicit channel ids (configs[0]: 3 and 17)
    decode_steps: int = 1
    rope_base: float = 10000.0

    @property
    def seed(self) -> int:
        return SEED0 + self.index

    @property
    def units(self) -> int:
        return self.n_layers * self.batch * self.n_heads

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


CONFIGS = {
    # configs[0]: tiny single head, fp32 N(0,1), channels 3 and 17 x20
    "cfg0_tiny": Workload("cfg0_tiny", 0, 1, 1, 1, 64, 256, "f32", "normal", 2, 20.0, (3, 17)),
    # configs[1]: ESM-2-650M single decode step, 33 x 20 heads, fp16 Student-t(4), 2 outlier channels x15
    "cfg1_650m_step": Workload("cfg1_650m_step", 1, 33, 1, 20, 64, 1024, "f16", "student_t4", 2, 15.0),
    # configs[2]: batch 32, 100 consecutive decode steps with tq_append (headline)
    "cfg2_650m_batch32": Workload("cfg2_650m_batch32", 2, 1, 32, 20, 64, 1024, "f16", "student_t4", 2, 15.0,
                                  decode_steps=100),
    # configs[3]: long context, fp16 N(0,1), 3 outlier channels x25
    "cfg3_long_splitk": Workload("cfg3_long_splitk", 3, 1, 4, 20, 64, 16384, "f16", "normal", 3, 25.0),
    # configs[4]: ESM-2-15B-shaped heads, d = 128, fp16 Student-t(4), no outliers stated
    "cfg4_15b_heads": Workload("cfg4_15b_heads", 4, 1, 8, 40, 128, 4096, "f16", "student_t4", 0, 1.0),
}


def _rng(w: Workload, stream: int) -> np.random.Generator:
    # independent named streams so that changing one tensor's size never shifts another's values
    return np.random.Generator(np.random.PCG64([w.seed, stream]))


def orthogonal_from_gaussian(rng: np.random.Generator, d: int) -> np.ndarray:
    """Q of QR(G), G ~ N(0,1)^{d x d}, columns sign-fixed so diag(R) > 0 (Haar-distributed)."""
    g = rng.standard_normal((d, d))
    q, r = np.linalg.qr(g)
    q = q * np.sign(np.diag(r))[None, :]
    return q.astype(np.float32)


def rotations(w: Workload):
    """(pi_k, pi_v): [L,H,d,d] fp32, one per (layer, head) (configs[1])."""
    rk, rv = _rng(w, 1), _rng(w, 2)
    L, H, d = w.n_layers, w.n_heads, w.head_dim
    pk = np.stack([orthogonal_from_gaussian(rk, d) for _ in range(L * H)]).reshape(L, H, d, d)
    pv = np.stack([orthogonal_from_gaussian(rv, d) for _ in range(L * H)]).reshape(L, H, d, d)
    return pk, pv


def sketch(w: Workload) -> np.ndarray:
    """S: [m,d] i.i.d. N(0,1), m = d (configs[0] 'a seeded Gaussian 64x64')."""
    return _rng(w, 3).standard_normal((w.head_dim, w.head_dim)).astype(np.float32)


def outlier_channels(w: Workload) -> np.ndarray:
    """[L,H,n_outlier] channel ids, fixed per head across tokens and batch."""
    L, H = w.n_layers, w.n_heads
    if w.n_outlier == 0:
        return np.zeros((L, H, 0), np.int64)
    if w.fixed_outliers:
        return np.broadcast_to(np.asarray(w.fixed_outliers, np.int64), (L, H, w.n_outlier)).copy()
    rng = _rng(w, 4)
    return np.stack([rng.choice(w.head_dim, size=w.n_outlier, replace=False) for _ in range(L * H)]).reshape(
        L, H, w.n_outlier)


def _draw(rng, w: Workload, shape):
    if w.dist == "normal":
        return rng.standard_normal(shape, dtype=np.float32)
    if w.dist == "student_t4":
        return rng.standard_t(4.0, size=shape).astype(np.float32)
    raise ValueError(w.dist)


def _np_dtype(w: Workload):
    return np.float16 if w.dtype == "f16" else np.float32


def layer_activations(w: Workload, layer: int, n_tokens: int | None = None, stream_base: int = 100):
    """(k, v) of one layer: [B,H,T,d] in the workload dtype, outlier channels scaled."""
    T = w.seq if n_tokens is None else n_tokens
    B, H, d = w.batch, w.n_heads, w.head_dim
    ch = outlier_channels(w)[layer]
    out = []
    for which in (0, 1):
        rng = _rng(w, stream_base + 2 * layer + which)
        x = _draw(rng, w, (B, H, T, d))
        for h in range(H):
            for c in ch[h]:
                x[:, h, :, c] *= w.outlier_scale
        out.append(x.astype(_np_dtype(w)))
    return out[0], out[1]


def layer_values_cold(w: Workload, layer: int, n_tokens: int | None = None):
    """Values of one layer as the paper describes them ("substantially colder ... kurtosis near 3.0"):
    plain N(0,1) per channel, no outlier channels, [B,H,T,d] in the workload dtype.  Used by the dual-LUT / shared-LUT
    ablation rows, where K and V must follow different distributions."""
    T = w.seq if n_tokens is None else n_tokens
    rng = _rng(w, 500_000 + layer)
    return rng.standard_normal((w.batch, w.n_heads, T, w.head_dim)).astype(_np_dtype(w))


def step_tokens(w: Workload, layer: int, step: int):
    """(q, k_new, v_new) of decode step `step` for one layer: each [B,H,d] in the workload dtype."""
    B, H, d = w.batch, w.n_heads, w.head_dim
    ch = outlier_channels(w)[layer]
    rng = _rng(w, 1_000_000 + 1000 * layer + step)
    out = []
    for _ in range(3):
        x = _draw(rng, w, (B, H, d))
        for h in range(H):
            for c in ch[h]:
                x[:, h, c] *= w.outlier_scale
        out.append(x.astype(_np_dtype(w)))
    return out[0], out[1], out[2]


def queries(w: Workload, layer: int):
    """q of the single decode query of one layer: [B,H,d]."""
    return step_tokens(w, layer, 999)[0]
