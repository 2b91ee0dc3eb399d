"""Pins of the oracle's decode attention and dense reference (Algorithm 1; Eq. 1; Eq. 4)."""
import math

import numpy as np
import pytest

from paper_2603_26110_b200 import workloads as W


def np_rope(x, pos, base=10000.0):
    """Independent RoPE (complex form of Eq. 2) for arrays [..., d] with a scalar or [...]-shaped position."""
    d = x.shape[-1]
    theta = base ** (-2.0 * np.arange(d // 2) / d)
    ang = np.asarray(pos, np.float64)[..., None] * theta
    z = (x[..., 0::2] + 1j * x[..., 1::2]) * np.exp(1j * ang)
    out = np.empty(x.shape, np.float64)
    out[..., 0::2], out[..., 1::2] = z.real, z.imag
    return out


def gauss_lut(oracle, d):
    return oracle.lloyd_max_gauss(1.0 / math.sqrt(d), 8)[0].astype(np.float32)


def make_case(oracle, B=2, H=3, T=40, d=64, seed=0):
    rng = np.random.default_rng(seed)
    haar = lambda: W.orthogonal_from_gaussian(rng, d)
    pi_k = np.stack([haar() for _ in range(H)])
    pi_v = np.stack([haar() for _ in range(H)])
    S = rng.standard_normal((d, d)).astype(np.float32)
    lut = gauss_lut(oracle, d)
    lut_k = np.tile(lut, (H, 1))
    lut_v = np.tile(lut * np.float32(1.1), (H, 1))  # a different V table exercises the dual-LUT path
    k = rng.standard_normal((B, H, T, d)).astype(np.float32)
    v = rng.standard_normal((B, H, T, d)).astype(np.float32)
    q = rng.standard_normal((B, H, d)).astype(np.float32)
    for x in (k, v, q):
        x[..., 3] *= 6
    return dict(pi_k=pi_k, pi_v=pi_v, S=S, lut_k=lut_k, lut_v=lut_v, k=k, v=v, q=q)


def test_dense_ref_matches_torch_sdpa(oracle):
    import torch

    c = make_case(oracle, B=2, H=2, T=33, seed=1)
    B, H, T, d = c["k"].shape
    q_pos = np.array([T - 1, T + 4], np.int32)
    seq = np.array([T, T - 7], np.int32)
    got = oracle.dense_attn_ref(c["q"], q_pos, seq, c["k"], c["v"])
    for b in range(B):
        t = seq[b]
        qr = np_rope(c["q"][b].astype(np.float64), q_pos[b])  # [H,d]
        kr = np_rope(c["k"][b, :, :t].astype(np.float64), np.broadcast_to(np.arange(t), (H, t)))
        want = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(qr)[:, None, :], torch.from_numpy(kr), torch.from_numpy(c["v"][b, :, :t].astype(np.float64)))
        assert np.allclose(got[b], want[:, 0, :].numpy(), atol=1e-12)


def test_decode_single_token_is_dequantised_value(oracle):
    # T = 1: softmax = 1, out = PI_V^T ( n_v * lut_V[codes_v] )
    c = make_case(oracle, B=1, H=2, T=1, seed=2)
    can = oracle.quantize_pack(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"])
    out = oracle.decode_attn(c["q"], [0], [1], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    for h in range(2):
        want = oracle.dequant_vector(can.v_codes[0, h, 0], can.v_norm[0, h, 0], c["pi_v"][h], c["lut_v"][h])
        assert np.allclose(out[0, h], want, atol=1e-12)
        # and the dequantised value approximates the original value (3-bit: ~0.19 relative error)
        rel = np.linalg.norm(want - c["v"][0, h, 0]) / np.linalg.norm(c["v"][0, h, 0])
        assert rel < 0.35


def test_decode_identical_keys_gives_mean_value(oracle):
    c = make_case(oracle, B=1, H=1, T=16, seed=3)
    # identical *post-RoPE* keys are not producible with positions 0..T-1, so use identical cache entries
    can = oracle.quantize_pack(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"])
    for plane in (can.k_codes, can.k_signs, can.k_norm, can.k_rnorm):
        plane[0, 0, :] = plane[0, 0, 0]
    out = oracle.decode_attn(c["q"], [15], [16], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    vs = np.stack([oracle.dequant_vector(can.v_codes[0, 0, t], can.v_norm[0, 0, t], c["pi_v"][0], c["lut_v"][0])
                   for t in range(16)])
    assert np.allclose(out[0, 0], vs.mean(axis=0), atol=1e-12)


def test_decode_equals_bruteforce_dense_attention_over_dequantised_cache(oracle):
    """north_star pin: brute-force dense attention on tiny inputs.  Without the sketch term the oracle must
    equal ordinary softmax attention between RoPE(q) and the *un-rotated* dequantised keys/values — this
    exercises Eq. 4 (PI moved from the keys to the query) and the final PI_V^T."""
    c = make_case(oracle, B=2, H=2, T=24, seed=4)
    B, H, T, d = c["k"].shape
    can = oracle.quantize_pack(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"])
    q_pos = np.array([T - 1, T - 1], np.int32)
    seq = np.array([T, T - 5], np.int32)
    got = oracle.decode_attn(c["q"], q_pos, seq, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can,
                             use_qjl=False)
    for b in range(B):
        for h in range(H):
            t = seq[b]
            kd = np.stack([oracle.dequant_vector(can.k_codes[b, h, j], can.k_norm[b, h, j], c["pi_k"][h], c["lut_k"][h])
                           for j in range(t)])  # ~ RoPE'd keys, un-rotated by PI_K^T
            vd = np.stack([oracle.dequant_vector(can.v_codes[b, h, j], can.v_norm[b, h, j], c["pi_v"][h], c["lut_v"][h])
                           for j in range(t)])
            s = kd @ np_rope(c["q"][b, h].astype(np.float64), q_pos[b]) / math.sqrt(d)
            p = np.exp(s - s.max())
            p /= p.sum()
            assert np.allclose(got[b, h], p @ vd, atol=1e-10)


def test_decode_qjl_term_matches_estimator(oracle):
    """With the sketch on, logit_j = n_j ( <q'', k_hat_j> + est_j ) / sqrt(d) where est_j is the pinned
    QJL estimator of <q'', r_j>; rebuilt here from quantize_vector's residual (|r| unrounded -> 1e-3 slack)."""
    c = make_case(oracle, B=1, H=1, T=12, seed=5)
    B, H, T, d = c["k"].shape
    can = oracle.quantize_pack(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"])
    got = oracle.decode_attn(c["q"], [T - 1], [T], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    q2 = c["pi_k"][0].astype(np.float64) @ np_rope(c["q"][0, 0].astype(np.float64), T - 1)
    lut = c["lut_k"][0].astype(np.float64)
    s = np.zeros(T)
    for j in range(T):
        r = oracle.quantize_vector(c["k"][0, 0, j], True, float(j), c["pi_k"][0], c["lut_k"][0], c["S"])
        khat = lut[r["codes"]]
        est = oracle.qjl_estimate(q2, r["u"] - khat, c["S"])
        n = oracle.f16_bits_to_f64(can.k_norm[0, 0, j])
        s[j] = n * (q2 @ khat + est) / math.sqrt(d)
    p = np.exp(s - s.max())
    p /= p.sum()
    vd = np.stack([oracle.dequant_vector(can.v_codes[0, 0, j], can.v_norm[0, 0, j], c["pi_v"][0], c["lut_v"][0])
                   for j in range(T)])
    assert np.allclose(got[0, 0], p @ vd, atol=2e-3 * np.abs(vd).max())
    # and the sketch term moves the logits towards the exact ones on average
    exact = np.array([q2 @ oracle.quantize_vector(c["k"][0, 0, j], True, float(j), c["pi_k"][0], c["lut_k"][0], c["S"])["u"]
                      for j in range(T)])


def test_qjl_correction_reduces_logit_error_on_average(oracle):
    rng = np.random.default_rng(6)
    d = 64
    lut = gauss_lut(oracle, d)
    Pi = W.orthogonal_from_gaussian(rng, d)
    S = rng.standard_normal((d, d)).astype(np.float32)
    e0 = e1 = 0.0
    for _ in range(300):
        k = rng.standard_normal(d)
        q2 = rng.standard_normal(d)
        r = oracle.quantize_vector(k, False, 0.0, Pi, lut, S)
        khat = lut.astype(np.float64)[r["codes"]]
        true = q2 @ r["u"]
        e0 += (q2 @ khat - true) ** 2
        # unbiased but noisy at m = d; its benefit is the removal of bias, so compare the means
        e1 += q2 @ khat + oracle.qjl_estimate(q2, r["u"] - khat, S) - true
    assert abs(e1 / 300) < 3 * math.sqrt(e0 / 300) / math.sqrt(300) * 2.0


def test_decode_ragged_and_empty(oracle):
    c = make_case(oracle, B=3, H=2, T=20, seed=7)
    can = oracle.quantize_pack(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"])
    seq = np.array([20, 0, 7], np.int32)
    out = oracle.decode_attn(c["q"], np.maximum(seq - 1, 0), seq, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    assert np.all(out[1] == 0.0) and np.all(np.isfinite(out))
    # entries beyond seq_len must not influence the result
    can.k_norm[2, :, 7:] = 0x7bff
    can.v_codes[2, :, 7:] = 0xff
    out2 = oracle.decode_attn(c["q"], np.maximum(seq - 1, 0), seq, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    assert np.array_equal(out, out2)


def test_quantised_attention_tracks_dense_attention_cfg0(oracle):
    """configs[0] end to end on the CPU: cosine of quantised decode attention vs exact fp64 attention.
    Reported next to the paper's >0.96 — a different quantity (final hidden state of a
    33-layer model on real proteins), so only a loose sanity bound is asserted: parity unpinned."""
    w = W.CONFIGS["cfg0_tiny"]
    pi_k, pi_v = W.rotations(w)
    S = W.sketch(w)
    lut = gauss_lut(oracle, w.head_dim)
    k, v = W.layer_activations(w, 0)
    q = W.queries(w, 0)
    luts = np.tile(lut, (w.n_heads, 1))
    can = oracle.quantize_pack(k, v, pi_k[0], pi_v[0], luts, luts, S, near_eps=1e-5)
    seq = np.array([w.seq], np.int32)
    out = oracle.decode_attn(q, seq - 1, seq, pi_k[0], pi_v[0], luts, luts, S, can)
    ref = oracle.dense_attn_ref(q, seq - 1, seq, k, v)
    cos = float((out * ref).sum() / (np.linalg.norm(out) * np.linalg.norm(ref)))
    assert cos > 0.85, cos
    # SURVEY 7 hard part 4: ~2.7e-4 of coordinates lie within 1e-5 of a threshold
    assert can.near_k.mean() < 5e-3


def test_workloads_are_seeded_and_shaped():
    w = W.CONFIGS["cfg1_650m_step"].scaled(n_layers=2, seq=64)
    k1, v1 = W.layer_activations(w, 1)
    k2, _ = W.layer_activations(w, 1)
    assert k1.dtype == np.float16 and k1.shape == (1, 20, 64, 64) and np.array_equal(k1, k2)
    ch = W.outlier_channels(w)
    assert ch.shape == (2, 20, 2)
    h = 5
    others = np.delete(np.arange(64), ch[1, h])
    assert np.abs(k1[0, h][:, ch[1, h]].astype(np.float32)).mean() > 5 * np.abs(k1[0, h][:, others].astype(np.float32)).mean()
    pk, pv = W.rotations(w)
    assert pk.shape == (2, 20, 64, 64) and not np.array_equal(pk[0, 0], pv[0, 0])
    assert np.abs(pk[1, 3].astype(np.float64).T @ pk[1, 3] - np.eye(64)).max() < 1e-6
    assert W.CONFIGS["cfg0_tiny"].fixed_outliers == (3, 17)
    assert W.CONFIGS["cfg4_15b_heads"].head_dim == 128 and W.CONFIGS["cfg3_long_splitk"].seq == 16384


# ------------------------------------------------------------------------------------------------ paper-literal Eq. 6-7 mode
def _literal_case(oracle, B=2, H=3, T=37, d=64, seed=11):
    """Raw-scale activations (|y| is NOT 1), LUT on the activation scale, S = I and PI_V = I as the paper has them."""
    rng = np.random.default_rng(seed)
    pi_k = np.stack([W.orthogonal_from_gaussian(rng, d) for _ in range(H)])
    pi_v = np.broadcast_to(np.eye(d, dtype=np.float32), (H, d, d)).copy()
    S = np.eye(d, dtype=np.float32)
    sig = np.array([0.7, 1.3, 2.1], np.float32)[:H]
    lut_k = np.stack([oracle.lloyd_max_gauss(float(s), 8)[0] for s in sig]).astype(np.float32)
    lut_v = np.stack([oracle.lloyd_max_gauss(float(1.5 * s), 8)[0] for s in sig]).astype(np.float32)
    k = (rng.standard_normal((B, H, T, d)) * sig[None, :, None, None]).astype(np.float32)
    v = (rng.standard_normal((B, H, T, d)) * 1.5 * sig[None, :, None, None]).astype(np.float32)
    q = rng.standard_normal((B, H, d)).astype(np.float32)
    ebar = np.array([0.21, 0.4, 0.66], np.float32)[:H]
    return dict(pi_k=pi_k, pi_v=pi_v, S=S, lut_k=lut_k, lut_v=lut_v, k=k, v=v, q=q, ebar=ebar, sig=sig)


def test_literal_mode_is_eq6_eq7_as_printed(oracle):
    """PAPER.md:170-179.  Per vector: codes = nearest LUT entry of the rotated activation itself (no normalisation),
    bits = sign(x - x^) (Eq. 6, S = I), norm plane = 1.0, rnorm plane decodes to e-bar m sqrt(2/pi).  And Eq. 7's claim
    "reducing the expected squared error by approximately e-bar^2 per element" is an identity when e-bar = mean |e|:
    mean (x - x~)^2 = mean e^2 - e-bar^2, checked on the reconstruction built from the oracle's own codes and bits."""
    c = _literal_case(oracle)
    d = 64
    rng = np.random.default_rng(5)
    x = rng.standard_normal(d) * 1.3
    h, pos = 1, 9
    out = oracle.quantize_vector_literal(x, True, pos, c["pi_k"][h], c["lut_k"][h], c["S"], float(c["ebar"][h]))
    y = c["pi_k"][h].astype(np.float64) @ np_rope(x, pos)
    assert np.allclose(out["y"], y, atol=1e-12)
    lut = c["lut_k"][h].astype(np.float64)
    want_codes = np.abs(y[:, None] - lut[None, :]).argmin(1)
    assert np.array_equal(out["codes"], want_codes)
    assert np.array_equal(out["bits"], (y - lut[want_codes] >= 0).astype(np.uint8))            # Eq. 6
    assert oracle.f16_bits_to_f64(out["norm_h"]) == 1.0
    g = oracle.f16_bits_to_f64(out["rnorm_h"])
    assert abs(g / (float(c["ebar"][h]) * d * math.sqrt(2 / math.pi)) - 1) <= 2.0 ** -11        # binary16 rounding only
    # values: no RoPE, no sketch, not normalised
    outv = oracle.quantize_vector_literal(x, False, pos, c["pi_v"][h], c["lut_v"][h], c["S"], 0.0)
    lv = c["lut_v"][h].astype(np.float64)
    assert np.array_equal(outv["codes"], np.abs(x[:, None] - lv[None, :]).argmin(1))
    # Eq. 7 error identity over many vectors, e-bar := the sample mean of |e|
    X = rng.standard_normal((400, d)) * float(c["sig"][h])
    E, S_, XH = [], [], []
    for xv in X:
        o = oracle.quantize_vector_literal(xv, True, 0.0, c["pi_k"][h], c["lut_k"][h], c["S"], 0.0)
        E.append(o["y"] - lut[o["codes"]]), S_.append(2.0 * o["bits"] - 1.0), XH.append(lut[o["codes"]])
    E, S_ = np.array(E), np.array(S_)
    ebar = np.abs(E).mean()
    assert abs(np.mean((E - S_ * ebar) ** 2) - (np.mean(E ** 2) - ebar ** 2)) < 1e-12
    assert np.mean((E - S_ * ebar) ** 2) < np.mean(E ** 2)


def test_literal_pack_indexing_and_decode_equals_attention_over_eq7_keys(oracle):
    """(a) tqo_quantize_pack_literal == the per-vector call with THAT head's PI / LUT / e-bar at position start_pos + t.
    (b) tqo_decode_attn over the literal planes == brute-force softmax attention over the Eq. 7 reconstruction
    k~ = lut_K[codes] + s e-bar (rotated back by PI_K^T) and v^ = lut_V[codes] (Algorithm 1 lines 6-11 with S = I)."""
    c = _literal_case(oracle)
    B, H, T, d = c["k"].shape
    sp = 5
    can = oracle.quantize_pack_literal(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], c["ebar"], start_pos=sp)
    for (b, h, t) in [(0, 0, 0), (1, 2, 36), (0, 1, 17)]:
        o = oracle.quantize_vector_literal(c["k"][b, h, t], True, sp + t, c["pi_k"][h], c["lut_k"][h], c["S"], float(c["ebar"][h]))
        assert np.array_equal(oracle.unpack_codes(can.k_codes[b, h, t], d), o["codes"])
        assert np.array_equal(oracle.unpack_bits(can.k_signs[b, h, t], d), o["bits"])
        assert can.k_norm[b, h, t] == o["norm_h"] and can.k_rnorm[b, h, t] == o["rnorm_h"]
        ov = oracle.quantize_vector_literal(c["v"][b, h, t], False, 0.0, c["pi_v"][h], c["lut_v"][h], c["S"], 0.0)
        assert np.array_equal(oracle.unpack_codes(can.v_codes[b, h, t], d), ov["codes"]) and can.v_norm[b, h, t] == ov["norm_h"]
    # (b) decode: the cache holds positions 0..T-1 when start_pos = 0
    can = oracle.quantize_pack_literal(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], c["ebar"])
    sl = np.full(B, T, np.int32)
    got = oracle.decode_attn(c["q"], sl - 1, sl, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    for b in range(B):
        for h in range(H):
            lk, lv = c["lut_k"][h].astype(np.float64), c["lut_v"][h].astype(np.float64)
            eb = oracle.f16_bits_to_f64(int(can.k_rnorm[b, h, 0])) * math.sqrt(math.pi / 2) / d  # e-bar as stored
            kt = np.stack([lk[oracle.unpack_codes(can.k_codes[b, h, t], d)] + (2.0 * oracle.unpack_bits(can.k_signs[b, h, t], d) - 1.0) * eb
                           for t in range(T)])                                   # Eq. 7, rotated basis
            vh = np.stack([lv[oracle.unpack_codes(can.v_codes[b, h, t], d)] for t in range(T)])
            q2 = c["pi_k"][h].astype(np.float64) @ np_rope(c["q"][b, h].astype(np.float64), T - 1)
            s = kt @ q2 / math.sqrt(d)
            p = np.exp(s - s.max())
            p /= p.sum()
            want = c["pi_v"][h].astype(np.float64).T @ (p @ vh)
            assert np.allclose(got[b, h], want, atol=1e-9)


# ------------------------------------------------------------------------------------------------ V-side residual sketch
def test_value_sketch_planes_and_decode_vq(oracle):
    """Algorithm 1 line 10, SURVEY.md 8(f) NEXT-1.  (a) The value planes are the key-side recipe without
    RoPE: bits = [S (u - lut[code]) >= 0], rnorm = |u - lut[code]|, rebuilt here with numpy.  (b) T = 1: out is the JL
    reconstruction PI_V^T n (lut_V[codes] + sqrt(pi/2)/m |r| S^T sigma).  (c) decode_attn_vq == brute-force softmax
    attention over those reconstructed values with the logits of the pinned decode_attn."""
    c = make_case(oracle, B=2, H=3, T=23, d=64, seed=4)
    B, H, T, d = c["k"].shape
    can = oracle.quantize_pack(c["k"], c["v"], c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"])
    oracle.add_value_sketch(can, c["v"], c["pi_v"], c["lut_v"], c["S"])
    cq = math.sqrt(math.pi / 2) / d

    def recon(b, h, t):  # rotated-basis JL reconstruction of value (b, h, t) from the stored planes
        lv = c["lut_v"][h].astype(np.float64)
        codes = oracle.unpack_codes(can.v_codes[b, h, t], d)
        sig = 2.0 * oracle.unpack_bits(can.v_signs[b, h, t], d) - 1.0
        n, g = oracle.f16_bits_to_f64(int(can.v_norm[b, h, t])), oracle.f16_bits_to_f64(int(can.v_rnorm[b, h, t]))
        return n * (lv[codes] + cq * g * (c["S"].astype(np.float64).T @ sig))

    for (b, h, t) in [(0, 0, 0), (1, 2, 22), (0, 1, 11)]:
        y = c["pi_v"][h].astype(np.float64) @ c["v"][b, h, t].astype(np.float64)
        u = y / np.linalg.norm(y)
        lv = c["lut_v"][h].astype(np.float64)
        r = u - lv[np.abs(u[:, None] - lv[None, :]).argmin(1)]
        assert np.array_equal(oracle.unpack_bits(can.v_signs[b, h, t], d), (c["S"].astype(np.float64) @ r >= 0).astype(np.uint8))
        assert abs(oracle.f16_bits_to_f64(int(can.v_rnorm[b, h, t])) / np.linalg.norm(r) - 1) <= 2.0 ** -11
    # (b) T = 1
    one = np.ones(B, np.int32)
    got1 = oracle.decode_attn_vq(c["q"], one - 1, one, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    for b in range(B):
        for h in range(H):
            assert np.allclose(got1[b, h], c["pi_v"][h].astype(np.float64).T @ recon(b, h, 0), atol=1e-12)
    # (c) full attention: weights from the pinned K side (decode_attn with V = one-hot trick is not needed: recompute the
    #     logits through decode_attn's own definition by probing with unit values) -> here simply by brute force
    sl = np.array([T, 9], np.int32)
    got = oracle.decode_attn_vq(c["q"], sl - 1, sl, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    base = oracle.decode_attn(c["q"], sl - 1, sl, c["pi_k"], c["pi_v"], c["lut_k"], c["lut_v"], c["S"], can)
    for b in range(B):
        for h in range(H):
            Tb = int(sl[b])
            q2 = c["pi_k"][h].astype(np.float64) @ np_rope(c["q"][b, h].astype(np.float64), Tb - 1)
            z = c["S"].astype(np.float64) @ q2
            lk = c["lut_k"][h].astype(np.float64)
            s = np.empty(Tb)
            for t in range(Tb):
                kc = oracle.unpack_codes(can.k_codes[b, h, t], d)
                sg = 2.0 * oracle.unpack_bits(can.k_signs[b, h, t], d) - 1.0
                n, g = oracle.f16_bits_to_f64(int(can.k_norm[b, h, t])), oracle.f16_bits_to_f64(int(can.k_rnorm[b, h, t]))
                s[t] = n * (q2 @ lk[kc] + cq * g * (z @ sg)) / math.sqrt(d)
            p = np.exp(s - s.max())
            p /= p.sum()
            vt = np.stack([recon(b, h, t) for t in range(Tb)])
            want = c["pi_v"][h].astype(np.float64).T @ (p @ vt)
            assert np.allclose(got[b, h], want, atol=1e-10)
            # and it differs from the K-only decode by exactly the sketch term
            lv = c["lut_v"][h].astype(np.float64)
            plain = np.stack([oracle.f16_bits_to_f64(int(can.v_norm[b, h, t])) * lv[oracle.unpack_codes(can.v_codes[b, h, t], d)] for t in range(Tb)])
            assert np.allclose(base[b, h], c["pi_v"][h].astype(np.float64).T @ (p @ plain), atol=1e-10)


def test_value_sketch_reconstruction_is_unbiased_over_S(oracle):
    """E_S[ sqrt(pi/2)/m |r| S^T sign(S r) ] = r (the vector form of the pinned inner-product estimator): Monte-Carlo over
    seeded Gaussian S, every coordinate within 4.5 standard errors, and the mean reconstruction error shrinks."""
    rng = np.random.default_rng(8)
    d = m = 64
    lut = gauss_lut(oracle, d)
    x = rng.standard_normal(d)
    u = x / np.linalg.norm(x)
    r = u - lut.astype(np.float64)[np.abs(u[:, None] - lut.astype(np.float64)[None, :]).argmin(1)]
    g = np.linalg.norm(r)
    n_draw = 4000
    acc, acc2 = np.zeros(d), np.zeros(d)
    for _ in range(n_draw):
        S = rng.standard_normal((m, d))
        est = math.sqrt(math.pi / 2) / m * g * (S.T @ np.where(S @ r >= 0, 1.0, -1.0))
        acc += est
        acc2 += est * est
    mean = acc / n_draw
    se = np.sqrt(np.maximum(acc2 / n_draw - mean ** 2, 1e-30) / n_draw)
    assert np.all(np.abs(mean - r) < 4.5 * se)
    assert np.linalg.norm(mean - r) < 0.1 * g
