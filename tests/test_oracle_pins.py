"""Pins of the CPU oracle (oracle/tq_oracle.c) against what the paper and the mathematics fix.

Each test checks an oracle function against something other than itself: closed forms, textbook tables
(tests/golden/), numpy/scipy library routines, brute force, Monte-Carlo.  No GPU is involved.
"""
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def haar(rng, d):
    q, r = np.linalg.qr(rng.standard_normal((d, d)))
    return (q * np.sign(np.diag(r))[None, :]).astype(np.float32)


# ---------------------------------------------------------------------------- binary16 conversion
def test_f16_roundtrip_matches_numpy(oracle):
    rng = np.random.default_rng(1)
    xs = np.concatenate([
        rng.uniform(0, 70000, 2000), rng.uniform(0, 1e-3, 2000), rng.uniform(0, 1e-7, 500),
        np.abs(rng.standard_normal(2000)) * 30,
        # exact ties between neighbouring binary16 values (round-to-even)
        np.array([1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11, 2048.0 + 1.0, 2048.0 + 3.0, 2.0 ** -25, 3 * 2.0 ** -25,
                  65504.0, 65519.9, 0.0, 2.0 ** -14, 2.0 ** -14 - 2.0 ** -25, 2.0 ** -24]),
    ])
    for x in xs:
        bits = oracle.f64_to_f16_bits(x)
        with np.errstate(over="ignore"):
            want = np.float16(min(x, 65504.0))  # the oracle clamps instead of overflowing (D6)
        assert bits == int(want.view(np.uint16)), (x, bits, int(want.view(np.uint16)))
        assert oracle.f16_bits_to_f64(bits) == float(want)


def test_f16_decode_all_finite_patterns(oracle):
    for h in list(range(0, 0x7c00, 7)) + [0x7bff, 0x0001, 0x03ff, 0x0400]:
        assert oracle.f16_bits_to_f64(h) == float(np.uint16(h).view(np.float16))


# ---------------------------------------------------------------------------- RoPE (Eq. 1-2)
def test_rope_closed_form_d2(oracle):
    # d = 2: theta_0 = base^0 = 1, so RoPE is the plane rotation by p radians (Eq. 2)
    p = 0.7
    out = oracle.rope(np.array([2.0, -1.0]), p)
    assert np.allclose(out, [2 * math.cos(p) + math.sin(p), 2 * math.sin(p) - math.cos(p)], atol=1e-15)


def test_rope_frequencies_and_complex_form(oracle):
    # theta_g = base^(-2g/d); pair (2g, 2g+1) is multiplied by exp(i p theta_g) (Eq. 2 as complex numbers)
    rng = np.random.default_rng(2)
    d, p, base = 8, 13.0, 10000.0
    x = rng.standard_normal(d)
    z = (x[0::2] + 1j * x[1::2]) * np.exp(1j * p * base ** (-2.0 * np.arange(d // 2) / d))
    want = np.empty(d)
    want[0::2], want[1::2] = z.real, z.imag
    assert np.allclose(oracle.rope(x, p, base, 0), want, atol=1e-13)
    # d = 4, base 1e4: theta_1 = 1e4^(-1/2) = 0.01
    out = oracle.rope(np.array([0.0, 0.0, 1.0, 0.0]), 50.0, 1e4, 0)
    assert np.allclose(out[2:], [math.cos(0.5), math.sin(0.5)], atol=1e-15)
    # half-split layout pairs (g, g + d/2)
    z2 = (x[: d // 2] + 1j * x[d // 2:]) * np.exp(1j * p * base ** (-2.0 * np.arange(d // 2) / d))
    assert np.allclose(oracle.rope(x, p, base, 1), np.concatenate([z2.real, z2.imag]), atol=1e-13)


def test_rope_invariants(oracle):
    rng = np.random.default_rng(3)
    d = 64
    q, k = rng.standard_normal(d), rng.standard_normal(d)
    assert np.array_equal(oracle.rope(q, 0.0), q)  # p = 0 is the identity
    assert abs(np.linalg.norm(oracle.rope(q, 917.0)) - np.linalg.norm(q)) < 1e-12  # orthogonal
    # <R_i q, R_j k> depends on j - i only
    a = oracle.rope(q, 5.0) @ oracle.rope(k, 12.0)
    b = oracle.rope(q, 105.0) @ oracle.rope(k, 112.0)
    c = q @ oracle.rope(k, 7.0)
    assert abs(a - b) < 1e-10 and abs(a - c) < 1e-10


def test_eq4_rotation_invariance(oracle):
    # north_star pins: PI^T PI = I to 1e-6; <PI R q, PI R k> = <R q, R k> to 1e-5 (Eq. 4)
    rng = np.random.default_rng(4)
    d = 64
    Pi = haar(rng, d)
    assert np.abs(Pi.T.astype(np.float64) @ Pi.astype(np.float64) - np.eye(d)).max() < 1e-6
    q, k = rng.standard_normal(d), rng.standard_normal(d)
    q[[3, 17]] *= 20
    k[[3, 17]] *= 20
    rq, rk = oracle.rope(q, 40.0), oracle.rope(k, 11.0)
    lhs = (Pi.astype(np.float64) @ rq) @ (Pi.astype(np.float64) @ rk)
    assert abs(lhs - rq @ rk) < 1e-5 * max(1.0, abs(rq @ rk))


# ---------------------------------------------------------------------------- Lloyd-Max (Eq. 5)
def _golden_lloyd():
    rows = {}
    with open(os.path.join(GOLDEN, "lloyd_max_gauss.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            lv, cs, ts, mse = [s.strip() for s in line.split("|")]
            rows[int(lv)] = ([float(x) for x in cs.split()], [float(x) for x in ts.split()], float(mse))
    return rows


@pytest.mark.parametrize("levels", [2, 4, 8])
def test_lloyd_max_gauss_matches_max1960_table(oracle, levels):
    cs, ts, mse = _golden_lloyd()[levels]
    c, t, m = oracle.lloyd_max_gauss(1.0, levels)
    pos_c = c[levels // 2:]
    pos_t = t[levels // 2:]  # t[levels/2 - 1] is the zero threshold
    assert np.allclose(pos_c, cs, rtol=6e-4), (pos_c, cs)
    assert np.allclose(pos_t, ts, rtol=6e-4), (pos_t, ts)
    assert abs(t[levels // 2 - 1]) < 1e-12
    assert abs(m - mse) < 6e-4 * mse * 10
    assert np.allclose(c, -c[::-1], atol=1e-12)  # symmetric


def test_lloyd_max_two_level_closed_form(oracle):
    c, t, m = oracle.lloyd_max_gauss(1.0, 2)
    assert abs(c[1] - math.sqrt(2 / math.pi)) < 1e-12 and abs(m - (1 - 2 / math.pi)) < 1e-12


def test_lloyd_max_fixed_point_by_quadrature(oracle):
    # centroid condition c_k = E[x | bin k] and boundary condition t_k = (c_k + c_{k+1})/2, the former
    # verified by numerical integration (independent of the oracle's closed-form truncated mean)
    from scipy import integrate

    sigma = 1.0 / 8.0  # N(0, 1/64), configs[0]
    c, t, mse = oracle.lloyd_max_gauss(sigma, 8)
    pdf = lambda x: math.exp(-0.5 * (x / sigma) ** 2) / (sigma * math.sqrt(2 * math.pi))
    edges = [-12 * sigma] + list(t) + [12 * sigma]
    total = 0.0
    for k in range(8):
        num = integrate.quad(lambda x: x * pdf(x), edges[k], edges[k + 1], epsabs=1e-14)[0]
        den = integrate.quad(pdf, edges[k], edges[k + 1], epsabs=1e-14)[0]
        assert abs(num / den - c[k]) < 1e-9
        total += integrate.quad(lambda x: (x - c[k]) ** 2 * pdf(x), edges[k], edges[k + 1], epsabs=1e-14)[0]
    assert np.allclose(t, 0.5 * (c[:-1] + c[1:]), atol=1e-14)
    assert abs(total / sigma ** 2 - mse) < 1e-8
    # scaling: N(0, sigma^2) solution = sigma x unit solution (+-0.030637 ... at d = 64)
    c1, _, _ = oracle.lloyd_max_gauss(1.0, 8)
    assert np.allclose(c, sigma * c1, atol=1e-15)
    assert abs(c[4] - 0.030637) < 2e-6 and abs(c[7] - 0.268993) < 2e-6


def test_lloyd_max_samples_is_kmeans_fixed_point(oracle):
    rng = np.random.default_rng(5)
    x = rng.standard_normal(400_000)
    c, mse = oracle.lloyd_max_samples(x, 8, iters=200)
    cg, _, mg = oracle.lloyd_max_gauss(1.0, 8)
    assert np.allclose(c, cg, atol=0.02) and abs(mse - mg) < 0.002
    # fixed point: every centroid is the mean of the samples nearest to it (numpy brute force)
    nearest = np.abs(x[:, None] - c[None, :]).argmin(axis=1)
    means = np.array([x[nearest == k].mean() for k in range(8)])
    assert np.allclose(means, c, atol=2e-3)
    assert abs(((x - c[nearest]) ** 2).mean() - mse) < 1e-6
    # an asymmetric distribution keeps its asymmetry (dual-LUT case)
    y = rng.gamma(2.0, 1.0, 100_000)
    cy, _ = oracle.lloyd_max_samples(y, 8)
    assert np.all(np.diff(cy) > 0) and cy[0] > 0


# ---------------------------------------------------------------------------- coding
def test_code_equals_bruteforce_argmin(oracle):
    rng = np.random.default_rng(6)
    c, t, _ = oracle.lloyd_max_gauss(1 / 8, 8)
    lut = c.astype(np.float32)
    us = np.concatenate([rng.standard_normal(3000) / 8, rng.uniform(-0.5, 0.5, 1000), [-1.0, 1.0, 0.0]])
    for u in us:
        thr = 0.5 * (lut[:-1] + lut[1:])  # fp32 midpoints
        if np.min(np.abs(u - thr.astype(np.float64))) < 1e-9:
            continue
        assert oracle.code(u, lut) == oracle.code_argmin(u, lut)
        assert oracle.code(u, lut) == int(np.abs(u - lut.astype(np.float64)).argmin())
    # tie on a threshold -> lower code (D7; first-minimum argmin)
    thr0 = float(np.float32(0.5) * (lut[3] + lut[4]))
    assert oracle.code(thr0, lut) == 3
    assert oracle.code(np.nextafter(thr0, 1.0), lut) == 4
    # an asymmetric LUT
    lut2 = np.array([-0.5, -0.2, -0.1, 0.0, 0.05, 0.1, 0.3, 0.9], np.float32)
    for u in rng.uniform(-1, 1, 2000):
        assert oracle.code(u, lut2) == int(np.abs(u - lut2.astype(np.float64)).argmin())


# ---------------------------------------------------------------------------- packing
def test_pack_matches_paper_snippet(oracle):
    rng = np.random.default_rng(7)
    shifts = np.arange(8) * 3
    for d in (8, 64, 128):
        for _ in range(50):
            idx = rng.integers(0, 8, size=(d // 8, 8))
            packed = (idx << shifts).sum(axis=-1)  # the paper's vectorised pack, verbatim semantics
            want = np.stack([(packed >> 0) & 0xff, (packed >> 8) & 0xff, (packed >> 16) & 0xff], axis=-1).astype(np.uint8)
            got = oracle.pack_codes(idx.reshape(-1))
            assert np.array_equal(got, want.reshape(-1))
            # the paper's unpack
            p32 = got.reshape(-1, 3).astype(np.uint32)
            p32 = p32[:, 0] | (p32[:, 1] << 8) | (p32[:, 2] << 16)
            assert np.array_equal((p32[:, None] >> shifts) & 0x7, idx)
            assert np.array_equal(oracle.unpack_codes(got, d), idx.reshape(-1))


def test_pack_roundtrip_exhaustive_small(oracle):
    # all 8^4 patterns in four positions of one 8-code group, other positions varying with the pattern
    for n in range(8 ** 4):
        codes = np.array([(n >> (3 * i)) & 7 for i in range(4)] + [(n * 5 + i) & 7 for i in range(4)], np.uint8)
        assert np.array_equal(oracle.unpack_codes(oracle.pack_codes(codes), 8), codes)
    # bit stream definition: bit (3i + b) of the LSB-first stream = bit b of code_i
    codes = np.zeros(64, np.uint8)
    codes[21] = 0b101
    stream = np.unpackbits(oracle.pack_codes(codes), bitorder="little")
    assert stream.sum() == 2 and stream[63] == 1 and stream[65] == 1


def test_sign_bit_packing(oracle):
    rng = np.random.default_rng(8)
    bits = rng.integers(0, 2, 64).astype(np.uint8)
    packed = oracle.pack_bits(bits)
    assert np.array_equal(np.unpackbits(packed, bitorder="little"), bits)
    assert np.array_equal(oracle.unpack_bits(packed, 64), bits)


# ---------------------------------------------------------------------------- per-vector quantizer
def _gauss_lut(oracle, d):
    return oracle.lloyd_max_gauss(1.0 / math.sqrt(d), 8)[0].astype(np.float32)


def test_quantize_vector_special_cases(oracle):
    d = 64
    lut = _gauss_lut(oracle, d)
    I = np.eye(d, dtype=np.float32)
    # x = 5 e_9, PI = I, S = I, value path: u = e_9 -> code 7 there, 0 elsewhere sits on the t = 0 tie -> 3
    x = np.zeros(d)
    x[9] = 5.0
    r = oracle.quantize_vector(x, False, 0.0, I, lut, I)
    assert r["codes"][9] == 7 and np.all(np.delete(r["codes"], 9) == 3)
    assert oracle.f16_bits_to_f64(r["norm_h"]) == 5.0
    # zero vector (D6): u = 0, norm 0
    r0 = oracle.quantize_vector(np.zeros(d), True, 3.0, I, lut, I)
    assert r0["norm_h"] == 0 and np.all(r0["codes"] == 3)
    # transposed-operand check: PI = permutation matrix P with (P x)_i = x_{perm[i]}
    rng = np.random.default_rng(9)
    perm = rng.permutation(d)
    P = np.zeros((d, d), np.float32)
    P[np.arange(d), perm] = 1.0
    x = rng.standard_normal(d)
    a = oracle.quantize_vector(x, False, 0.0, P, lut, I)
    b = oracle.quantize_vector(x, False, 0.0, I, lut, I)
    assert np.array_equal(a["codes"], b["codes"][perm])
    # keys get RoPE, values do not
    k5 = oracle.quantize_vector(x, True, 5.0, I, lut, I)
    k5b = oracle.quantize_vector(oracle.rope(x, 5.0), True, 0.0, I, lut, I)
    v5 = oracle.quantize_vector(x, False, 5.0, I, lut, I)
    assert np.array_equal(k5["codes"], k5b["codes"]) and np.array_equal(v5["codes"], b["codes"])


def test_quantize_vector_scale_invariance_and_norm(oracle):
    rng = np.random.default_rng(10)
    d = 64
    lut = _gauss_lut(oracle, d)
    Pi, S = haar(rng, d), rng.standard_normal((d, d)).astype(np.float32)
    x = rng.standard_normal(d)
    a = oracle.quantize_vector(x, True, 7.0, Pi, lut, S)
    b = oracle.quantize_vector(4.0 * x, True, 7.0, Pi, lut, S)  # power of two: exact in fp64
    assert np.array_equal(a["codes"], b["codes"]) and np.array_equal(a["bits"], b["bits"])
    assert a["rnorm_h"] == b["rnorm_h"]
    assert oracle.f16_bits_to_f64(b["norm_h"]) == 4.0 * oracle.f16_bits_to_f64(a["norm_h"])
    # the stored norm is |PI R x| = |x| (orthogonal maps), rounded to binary16
    assert a["norm_h"] == int(np.float16(np.linalg.norm(x)).view(np.uint16))
    assert abs(np.linalg.norm(a["u"]) - 1.0) < 1e-12


def test_residual_sketch_reduces_to_paper_eq6_when_S_is_identity(oracle):
    # Eq. 6: s = sign(x - x_hat) per element  ==  sign(S r) with S = I
    rng = np.random.default_rng(11)
    d = 64
    lut = _gauss_lut(oracle, d)
    Pi = haar(rng, d)
    I = np.eye(d, dtype=np.float32)
    x = rng.standard_normal(d)
    r = oracle.quantize_vector(x, True, 2.0, Pi, lut, I)
    resid = r["u"] - lut.astype(np.float64)[r["codes"]]
    assert np.array_equal(r["bits"], (resid >= 0).astype(np.uint8))
    assert r["rnorm_h"] == int(np.float16(np.linalg.norm(resid)).view(np.uint16))
    # S = permutation rows: bit_j = sign(r_{perm[j]}) (catches a transposed S)
    perm = rng.permutation(d)
    Sp = np.zeros((d, d), np.float32)
    Sp[np.arange(d), perm] = 1.0
    rp = oracle.quantize_vector(x, True, 2.0, Pi, lut, Sp)
    assert np.array_equal(rp["bits"], r["bits"][perm])


def test_quantizer_mse_matches_lloyd_max_theory(oracle):
    # Haar-rotated unit vectors have ~N(0, 1/d) coordinates: E|u - u_hat|^2 ~ 0.0345 (Max 1960, 8 levels)
    rng = np.random.default_rng(12)
    d = 64
    lut = _gauss_lut(oracle, d)
    Pi, I = haar(rng, d), np.eye(d, dtype=np.float32)
    errs = []
    for _ in range(400):
        x = rng.standard_normal(d)
        x[[3, 17]] *= 20  # outlier channels are spread by the rotation
        r = oracle.quantize_vector(x, False, 0.0, Pi, lut, I)
        errs.append(np.sum((r["u"] - lut.astype(np.float64)[r["codes"]]) ** 2))
    assert abs(np.mean(errs) - 0.03454) < 0.004, np.mean(errs)
    # without the rotation the same vectors quantise far worse ("No PI rotation")
    errs_id = []
    for _ in range(200):
        x = rng.standard_normal(d)
        x[[3, 17]] *= 20
        r = oracle.quantize_vector(x, False, 0.0, I, lut, I)
        errs_id.append(np.sum((r["u"] - lut.astype(np.float64)[r["codes"]]) ** 2))
    assert np.mean(errs_id) > 3 * np.mean(errs)


# ---------------------------------------------------------------------------- QJL estimator (D2)
def test_qjl_estimator_unbiased_monte_carlo(oracle):
    rng = np.random.default_rng(13)
    d = m = 64
    q = rng.standard_normal(d) * 3
    r = rng.standard_normal(d) * 0.02
    true = float(q @ r)
    n = 20000
    est = np.array([oracle.qjl_estimate(q, r, rng.standard_normal((m, d)).astype(np.float32)) for _ in range(n)])
    se = est.std(ddof=1) / math.sqrt(n)
    assert abs(est.mean() - true) < 4 * se, (est.mean(), true, se)
    bound = (math.pi / 2) / m * (q @ q) * (r @ r)
    assert est.var() < 1.05 * bound
    # q parallel to r: expectation |q||r|
    est2 = np.array([oracle.qjl_estimate(5 * r, r, rng.standard_normal((m, d)).astype(np.float32)) for _ in range(4000)])
    assert abs(est2.mean() - 5 * (r @ r)) < 4 * est2.std(ddof=1) / math.sqrt(4000)
    # a wrong constant (e.g. sqrt(2/pi) instead of sqrt(pi/2)) would be off by a factor pi/2
    assert abs(est.mean() / true - 1.0) < 0.25


# ---------------------------------------------------------------------------- memory accounting (Table 4)
def test_memory_accounting_against_paper_table4():
    vals = {}
    with open(os.path.join(GOLDEN, "paper_table4_memory.txt")) as f:
        for line in f:
            if not line.startswith("#") and line.strip():
                k, v = line.split()
                vals[k] = float(v)
    MiB = 2.0 ** 20
    elems = 2 * 33 * 20 * 64 * 1024  # Eq. 3
    assert abs(elems * 4 / MiB - vals["fp32_kv_cache"]) < 0.05
    # the paper's INT32 container holds 8 codes: 4 bit / element
    assert abs(elems * 4 / 8 / MiB - vals["packed_k_v"]) < 0.1
    # sign bits for K only (D3)
    assert abs(elems / 2 / 8 / MiB - vals["qjl_signs"]) < 0.1
    assert abs(vals["fp32_kv_cache"] / vals["total"] - vals["ratio"]) < 0.05
    # ours: 62 B per cached token-head at d = 64 (24 + 8 + 2 + 2 for K, 24 + 2 for V)
    ours = 33 * 20 * 1024 * 62 / MiB
    assert abs(ours - 40.0) < 0.1 and ours < vals["total"]


# ---------------------------------------------------------------------------- whole-layer indexing
def test_quantize_pack_start_pos_and_per_head_indexing(oracle):
    """tqo_quantize_pack(start_pos = s) must equal tqo_quantize_vector(pos = s + t) plane by plane, with THAT head's PI and
    LUT (pins the start_pos offset of the RoPE position and the pi + h d d / lut + 8 h indexing at B, H > 1;
    SURVEY.md §8(c) steps 1-6).  The per-vector call is pinned on its own above."""
    rng = np.random.default_rng(2603)
    B, H, T, d, s = 2, 3, 5, 64, 7
    pi_k = np.stack([haar(rng, d) for _ in range(H)])
    pi_v = np.stack([haar(rng, d) for _ in range(H)])
    lut0 = oracle.lloyd_max_gauss(1 / 8, 8)[0].astype(np.float32)
    lut_k = np.sort(np.stack([lut0 * np.float32(1 + 0.07 * h) for h in range(H)]), axis=-1)
    lut_v = np.sort(np.stack([lut0 * np.float32(1.3 - 0.05 * h) for h in range(H)]), axis=-1)
    S = rng.standard_normal((d, d)).astype(np.float32)
    k = rng.standard_normal((B, H, T, d)).astype(np.float32)
    v = rng.standard_normal((B, H, T, d)).astype(np.float32)
    k[..., 3] *= 20
    can = oracle.quantize_pack(k, v, pi_k, pi_v, lut_k, lut_v, S, start_pos=s)
    again0 = oracle.quantize_pack(k, v, pi_k, pi_v, lut_k, lut_v, S, start_pos=0)
    assert not np.array_equal(can.k_codes, again0.k_codes)  # the position matters for keys ...
    assert np.array_equal(can.v_codes, again0.v_codes)      # ... and not for values (no RoPE on V)
    for b in range(B):
        for h in range(H):
            for t in range(T):
                qk = oracle.quantize_vector(k[b, h, t], True, s + t, pi_k[h], lut_k[h], S)
                qv = oracle.quantize_vector(v[b, h, t], False, 0, pi_v[h], lut_v[h], S)
                assert np.array_equal(oracle.unpack_codes(can.k_codes[b, h, t], d), qk["codes"]), (b, h, t)
                assert np.array_equal(oracle.unpack_bits(can.k_signs[b, h, t], d), qk["bits"]), (b, h, t)
                assert can.k_norm[b, h, t] == qk["norm_h"] and can.k_rnorm[b, h, t] == qk["rnorm_h"]
                assert np.array_equal(oracle.unpack_codes(can.v_codes[b, h, t], d), qv["codes"]), (b, h, t)
                assert can.v_norm[b, h, t] == qv["norm_h"]
    # a wrong head's matrices or table would not reproduce the planes
    wrong = oracle.quantize_vector(k[1, 2, 4], True, s + 4, pi_k[1], lut_k[2], S)
    assert not np.array_equal(oracle.unpack_codes(can.k_codes[1, 2, 4], d), wrong["codes"])


def test_key_sketch_values_are_S_times_the_residual(oracle):
    """tqo_key_sketch_values returns (S r)_j: rebuilt here with numpy from the per-vector call's unit vector and codes,
    and its signs are the stored sign bits (>= 0 -> 1, D7).  The GPU parity tests use it to show that a sign
    mismatch can only sit where |(S r)_j| is at rounding level."""
    rng = np.random.default_rng(77)
    d = 64
    Pi = haar(rng, d)
    S = rng.standard_normal((d, d)).astype(np.float32)
    lut = oracle.lloyd_max_gauss(1 / 8, 8)[0].astype(np.float32)
    for pos in (0, 5, 1023):
        x = rng.standard_normal(d).astype(np.float32)
        x[17] *= 20
        qv = oracle.quantize_vector(x, True, pos, Pi, lut, S)
        sr = oracle.key_sketch_values(x, pos, Pi, lut, S)
        r = qv["u"] - lut[qv["codes"]].astype(np.float64)
        assert np.allclose(sr, S.astype(np.float64) @ r, rtol=0, atol=1e-12)
        assert np.array_equal((sr >= 0).astype(np.uint8), qv["bits"])
        assert abs(np.linalg.norm(r) - oracle.f16_bits_to_f64(qv["rnorm_h"])) <= 2.0 ** -11 * np.linalg.norm(r) + 1e-12


# ---------------------------------------------------------------------------- the tolerance band (near_k / near_v)
def _planted_unit_vector(rng, th, plan, d):
    """fp64 unit vector whose coordinate i equals th[q] + delta for (i, q, delta) in plan; the other coordinates are random
    and scaled so that the norm is exactly 1."""
    u = np.zeros(d)
    for i, q, delta in plan:
        u[i] = float(th[q]) + delta
    free = np.array([i for i in range(d) if i not in {p[0] for p in plan}])
    r = rng.standard_normal(free.size)
    u[free] = r * math.sqrt((1.0 - (u ** 2).sum()) / (r ** 2).sum())
    assert abs(np.linalg.norm(u) - 1.0) < 1e-14
    return u


def test_tolerance_band_marks_exactly_the_coordinates_within_eps_of_a_threshold(oracle):
    """north_star: codes are bit-exact "except coordinates within 1e-5 of a decision boundary".  near_k / near_v of
    tqo_quantize_pack decide which mismatches the GPU tests forgive, so the band itself is pinned here: unit coordinates
    are PLANTED at threshold +- 0.5e-5 (must be marked) and threshold +- 2e-5 (must not be), per head with that head's own
    LUT, behind a permutation PI for the values (the mask is indexed by the ROTATED coordinate).  A band ten times too
    wide, a band taken on the un-normalised vector, the other head's LUT or an un-permuted index each fail."""
    d, H = 64, 2
    eps = 1e-5
    lut0 = oracle.lloyd_max_gauss(1.0 / math.sqrt(d), 8)[0].astype(np.float32)
    luts = np.stack([lut0, (lut0 * np.float32(0.8)).astype(np.float32)])
    th = np.stack([(np.float32(0.5) * (l[:-1] + l[1:])).astype(np.float32) for l in luts])  # [H, 7] fp32, as the method rounds them
    plan = [(0, 1, +0.5e-5), (1, 4, -0.5e-5), (2, 5, +2e-5), (3, 2, -2e-5), (4, 3, +0.9e-5), (5, 0, -1.1e-5)]
    marked, unmarked = [0, 1, 4], [2, 3, 5]
    rng = np.random.default_rng(2603)
    perm = rng.permutation(d)
    inv = np.argsort(perm)
    P = np.zeros((d, d), np.float32)
    P[np.arange(d), perm] = 1.0  # y[i] = x[perm[i]]
    eye = np.eye(d, dtype=np.float32)
    k = np.zeros((1, H, 1, d), np.float32)
    v = np.zeros((1, H, 1, d), np.float32)
    for h in range(H):
        uk = _planted_unit_vector(rng, th[h], plan, d)
        uv = _planted_unit_vector(rng, th[h], plan, d)
        k[0, h, 0] = (uk * 3.7).astype(np.float32)        # position 0: RoPE is the identity, PI_K = I
        v[0, h, 0] = (uv * 0.41).astype(np.float32)[inv]  # PI_V = P brings coordinate i of uv back to slot i
    S = rng.standard_normal((d, d)).astype(np.float32)
    can = oracle.quantize_pack(k, v, np.stack([eye, eye]), np.stack([P, P]), luts, luts, S, near_eps=eps)
    for h in range(H):
        for name, near, x in (("k", can.near_k, k[0, h, 0].astype(np.float64)), ("v", can.near_v, v[0, h, 0].astype(np.float64)[perm])):
            got = near[0, h, 0].astype(bool)
            assert all(got[i] for i in marked), (name, h, got[:6])
            assert not any(got[i] for i in unmarked), (name, h, got[:6])
            # ... and nothing else: the definition written out in numpy on the same fp32 inputs
            u = x / np.linalg.norm(x)
            want = (np.abs(u[:, None] - th[h].astype(np.float64)[None, :]) < eps).any(axis=1)
            assert np.array_equal(got, want), (name, h)
            assert got.sum() == len(marked)
    # the other head's thresholds would not do: head 1's coordinates planted on non-zero thresholds are far from head 0's
    u1 = k[0, 1, 0].astype(np.float64) / np.linalg.norm(k[0, 1, 0].astype(np.float64))
    assert not (np.abs(u1[[0, 1], None] - th[0].astype(np.float64)[None, :]) < 10 * eps).any()


def test_tolerance_band_of_the_paper_literal_mode_scales_with_the_vector_norm(oracle):
    """DESIGN.md section 2, reading D17: in the paper-literal mode the coded coordinates are not normalised, so the band is
    near_eps x max(1, |y|).  Planted on y itself: |y| = 5 -> band 5e-5 (a coordinate 2.5e-5 from a threshold is marked,
    one 1e-4 away is not); |y| = 0.5 -> band stays 1e-5 (0.7e-5 marked, 2e-5 not)."""
    d, H = 64, 1
    eps = 1e-5
    lut = (oracle.lloyd_max_gauss(1.0 / math.sqrt(d), 8)[0] * 4.0).astype(np.float32)[None]
    th = (np.float32(0.5) * (lut[0, :-1] + lut[0, 1:])).astype(np.float32)
    rng = np.random.default_rng(7)
    eye = np.eye(d, dtype=np.float32)[None]

    def planted(norm, plan):
        y = np.zeros(d)
        for i, q, delta in plan:
            y[i] = float(th[q]) + delta
        free = np.arange(len(plan), d)
        r = rng.standard_normal(free.size)
        y[free] = r * math.sqrt((norm ** 2 - (y ** 2).sum()) / (r ** 2).sum())
        return y.astype(np.float32)

    big = planted(5.0, [(0, 1, +2.5e-5), (1, 5, -2.5e-5), (2, 3, +1e-4), (3, 2, -1e-4)])
    small = planted(0.5, [(0, 3, +0.7e-5), (1, 4, -0.7e-5), (2, 2, +2e-5), (3, 3, -2e-5)])
    k = np.stack([big, small])[None, None]  # [1, 1, 2, d]: two tokens ... position 1 would rotate the second: use v
    can = oracle.quantize_pack_literal(np.zeros_like(k), k, eye, eye, lut, lut, np.eye(d, dtype=np.float32),
                                       np.array([0.01], np.float32), near_eps=eps)
    for t, x in enumerate((big, small)):
        got = can.near_v[0, 0, t].astype(bool)
        assert got[0] and got[1] and not got[2] and not got[3], (t, got[:4])
        y = x.astype(np.float64)
        band = eps * max(1.0, float(np.linalg.norm(y)))
        want = (np.abs(y[:, None] - th.astype(np.float64)[None, :]) < band).any(axis=1)
        assert np.array_equal(got, want) and got.sum() == 2
    # keys at position 0 (RoPE = identity) take the same band
    can_k = oracle.quantize_pack_literal(big[None, None, None], np.zeros((1, 1, 1, d), np.float32), eye, eye, lut, lut,
                                         np.eye(d, dtype=np.float32), np.array([0.01], np.float32), near_eps=eps)
    assert np.array_equal(can_k.near_k[0, 0, 0], can.near_v[0, 0, 0])
