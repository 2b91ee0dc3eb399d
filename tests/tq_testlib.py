"""Helpers shared by the GPU parity tests: build seeded cases, run both sides, compare with the
north_star tolerances (BASELINE.json): codes/sign bits bit-exact except coordinates within 1e-5 of a
decision boundary (mismatch fraction <= 1e-4), attention outputs max-abs <= 2e-3 and cosine >= 0.9999 on
identical cache bytes."""
from __future__ import annotations

import math

import numpy as np

from paper_2603_26110_b200 import workloads as W

NEAR_EPS = 1e-5
MAX_MISMATCH_FRAC = 1e-4
OUT_MAX_ABS = 2e-3
OUT_MIN_COS = 0.9999
# Stored binary16 norms ("norm rule"): north_star states no norm tolerance.  A kernel that computes
# the norm in fp32 (relative error e <= about 5e-7: two-term fp16 products, fp32 accumulation of d terms, fp32 sqrt) rounds
# to a different binary16 than the fp64 oracle only when the exact value lies within e n of a rounding tie; ties are
# 2^-11 .. 2^-10 apart relative to n, so that happens to at most about 2 e 2^11 = 2e-3 of the entries and never by more
# than one ulp.  One entry is always allowed (small cases hold a few hundred norms).  Two fp32 kernels compared with
# each other (the tensor-core and the CUDA-core quantize kernels) each carry their own e: twice the rate.
NORM_MAX_ULP = 1
NORM_ULP_RATE = 2e-3


def assert_norm_ulps(a, b, what="", fp32_sides: int = 1):
    """a, b: binary16 bit patterns (any integer dtype / view) of the same norms from two implementations."""
    dd = np.abs(np.asarray(a).astype(np.int32) - np.asarray(b).astype(np.int32))
    rate = float((dd > 0).mean()) if dd.size else 0.0
    assert dd.max(initial=0) <= NORM_MAX_ULP, (what, int(dd.max(initial=0)))
    assert rate <= fp32_sides * NORM_ULP_RATE + 1.0 / max(1, dd.size), (what, rate)
    return rate


def make_arrays(oracle, w: W.Workload, rope_cs, lut_scale_v: float = 1.0, per_head_lut: bool = False):
    """Calibration arrays as DATA for both sides: PI/S from the seeded generators, LUT from the oracle's
    Lloyd-Max on N(0, 1/d) (configs[0]); lut_scale_v != 1 makes the V table differ (dual-LUT path).
    rope_cs is the product's own table (tq_calibrate_host); the oracle evaluates RoPE itself in fp64."""
    pi_k, pi_v = W.rotations(w)
    S = W.sketch(w)
    lut = oracle.lloyd_max_gauss(1.0 / math.sqrt(w.head_dim), 8)[0].astype(np.float32)
    L, H = w.n_layers, w.n_heads
    lut_k = np.tile(lut, (L, H, 1))
    lut_v = np.tile(lut * np.float32(lut_scale_v), (L, H, 1))
    if per_head_lut:  # slightly different tables per head
        rng = np.random.default_rng(w.seed + 77)
        lut_k = np.sort(lut_k * (1 + 0.05 * rng.standard_normal(lut_k.shape)).astype(np.float32), axis=-1)
        lut_v = np.sort(lut_v * (1 + 0.05 * rng.standard_normal(lut_v.shape)).astype(np.float32), axis=-1)
    return dict(pi_k=pi_k, pi_v=pi_v, lut_k=lut_k, lut_v=lut_v, S=S, rope_cs=rope_cs)


def canonical_to_numpy(planes: dict):
    return {k: v.cpu().numpy() for k, v in planes.items()}


def unpack_codes_np(packed: np.ndarray, d: int) -> np.ndarray:
    """[..., 3d/8] bytes -> [..., d] codes (vectorised restatement of the canonical bit stream, test-side)."""
    bits = np.unpackbits(packed, axis=-1, bitorder="little")
    bits = bits.reshape(*packed.shape[:-1], d, 3)
    return (bits[..., 0] | (bits[..., 1] << 1) | (bits[..., 2] << 2)).astype(np.uint8)


def compare_quantize(can_oracle, gpu: dict, d: int, what: str = ""):
    """Returns a report dict; asserts the north_star quantize tolerances."""
    rep = {}
    for side, codes_key, near in (("k", "k_codes", can_oracle.near_k), ("v", "v_codes", can_oracle.near_v)):
        co = unpack_codes_np(getattr(can_oracle, codes_key), d)
        cg = unpack_codes_np(gpu[codes_key], d)
        diff = co != cg
        # every mismatch must sit inside the 1e-5 band around a threshold, and differ by one level
        assert not np.any(diff & (near == 0)), f"{what}: {side} code mismatch away from a decision boundary"
        assert np.all(np.abs(co.astype(int) - cg.astype(int))[diff] == 1)
        rep[f"{side}_code_mismatch_frac"] = float(diff.mean())
        assert diff.mean() <= MAX_MISMATCH_FRAC, (what, side, diff.mean())
        rep[f"{side}_vec_equal"] = ~diff.any(axis=-1)
    # sign bits: only on key vectors whose codes agree (a flipped code changes r)
    ok = rep["k_vec_equal"]
    so = np.unpackbits(can_oracle.k_signs, axis=-1, bitorder="little")
    sg = np.unpackbits(gpu["k_signs"], axis=-1, bitorder="little")
    sdiff = (so != sg) & ok[..., None]
    rep["sign_mismatch_frac"] = float(sdiff.sum() / max(1, ok.sum() * so.shape[-1]))
    assert rep["sign_mismatch_frac"] <= MAX_MISMATCH_FRAC, (what, rep["sign_mismatch_frac"])
    # norms: binary16 of an fp32 vs an fp64 norm may differ by one ulp when the value sits on a rounding tie
    for name, mask in (("k_norm", None), ("k_rnorm", ok), ("v_norm", None)):
        a = getattr(can_oracle, name).astype(np.int32)
        b = gpu[name].view(np.uint16).astype(np.int32)
        if mask is not None:  # |r| is only comparable where the codes agree
            a, b = a[mask], b[mask]
        rep[f"{name}_ulp_mismatch_frac"] = assert_norm_ulps(a, b, f"{what} {name}")
    del rep["k_vec_equal"], rep["v_vec_equal"]
    return rep


def compare_outputs(out_gpu: np.ndarray, out_oracle: np.ndarray, what: str = "", max_abs=OUT_MAX_ABS):
    a = out_gpu.astype(np.float64).ravel()
    b = out_oracle.ravel()
    err = float(np.abs(a - b).max(initial=0.0))
    den = np.linalg.norm(a) * np.linalg.norm(b)
    cos = float(a @ b / den) if den > 0 else 1.0
    assert np.all(np.isfinite(a)), what
    assert err <= max_abs, (what, err)
    assert cos >= OUT_MIN_COS, (what, cos)
    return dict(max_abs=err, cosine=cos)


def to_torch_canonical(can, device="cuda"):
    import torch

    return dict(k_codes=torch.from_numpy(can.k_codes).to(device), k_signs=torch.from_numpy(can.k_signs).to(device),
                k_norm=torch.from_numpy(can.k_norm.view(np.int16)).to(device),
                k_rnorm=torch.from_numpy(can.k_rnorm.view(np.int16)).to(device),
                v_codes=torch.from_numpy(can.v_codes).to(device),
                v_norm=torch.from_numpy(can.v_norm.view(np.int16)).to(device))
