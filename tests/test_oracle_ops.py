"""Pins for the oracle's single operations: closed forms, special cases and library routines
(SURVEY.md §8(c) C-3 "O-AR decoder math" (ii)).  CPU only."""
import math
import os

import numpy as np
import pytest
import torch

import oracle as ora
import spd_inputs as si

GOLD = os.path.join(os.path.dirname(__file__), "golden")
rng = np.random.default_rng(0)


def bf16(x):
    return si.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def test_bf16_rounding_is_rne_like_torch():
    x = rng.standard_normal(20000).astype(np.float32) * 3
    # exact ties and neighbours: mantissa tail 0x8000 (tie), 0x7fff, 0x8001, odd/even kept bit
    ties = np.array([0x3F808000, 0x3F818000, 0x3F807FFF, 0x3F808001, 0xBF808000, 0x00008000, 0x7F7F7FFF],
                    dtype=np.uint32).view(np.float32)
    x = np.concatenate([x, ties])
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = np.array([ora.op_f32_to_bf16(float(v)) for v in x], dtype=np.uint16)
    assert np.array_equal(got, want)
    # and the generator's own rounding (used to make the weights) agrees with both
    assert np.array_equal(si.f32_to_bf16_bits(x), want)


def test_splitmix64_known_vectors():
    # tests/golden/splitmix64.txt: first outputs of the public-domain SplitMix64 generator, state 0
    rows = [l.split() for l in open(os.path.join(GOLD, "splitmix64.txt")) if l.strip() and not l.startswith("#")]
    gamma = 0x9E3779B97F4A7C15
    for i, (_, want) in enumerate(rows):
        assert ora.op_splitmix64((i * gamma) & (2 ** 64 - 1)) == int(want, 16)


def test_rmsnorm_constant_vector_and_scale_invariance():
    d = 96
    g = bf16(rng.uniform(0.5, 1.5, d))
    gf = si.bf16_bits_to_f32(g)
    for c in (3.0, -0.25):
        out = ora.op_rmsnorm(np.full(d, c, np.float32), g, 0.0)
        np.testing.assert_allclose(out, math.copysign(1.0, c) * gf, rtol=1e-6)
    x = rng.standard_normal(d).astype(np.float32)
    a = ora.op_rmsnorm(x, g, 0.0)
    b = ora.op_rmsnorm(4 * x, g, 0.0)
    np.testing.assert_allclose(a, b, rtol=1e-6)
    # definition with eps, float64
    eps = 1e-6
    want = x.astype(np.float64) / np.sqrt(np.mean(x.astype(np.float64) ** 2) + np.float32(eps)) * gf
    np.testing.assert_allclose(ora.op_rmsnorm(x, g, eps), want, rtol=1e-6)


def test_gemv_matches_float64_matmul_and_is_not_transposed():
    rows, k = 37, 203  # ragged: k not a multiple of 16
    w = bf16(rng.standard_normal((rows, k)) * 0.05)
    x = rng.standard_normal(k).astype(np.float32)
    want = si.bf16_bits_to_f32(w).astype(np.float64) @ x.astype(np.float64)
    np.testing.assert_allclose(ora.op_gemv(w, x), want, rtol=2e-6, atol=1e-7)
    # one-hot input selects a column
    e = np.zeros(k, np.float32)
    e[5] = 1
    assert np.array_equal(ora.op_gemv(w, e), si.bf16_bits_to_f32(w)[:, 5])


def test_rope_identity_norm_composition_and_closed_form():
    H, hd, base = 3, 16, 1e6
    v = rng.standard_normal(H * hd).astype(np.float32)
    assert np.array_equal(ora.op_rope(v, H, hd, 0, base), v)            # pos 0 is the identity
    r = ora.op_rope(v, H, hd, 1234, base).reshape(H, hd)
    vv = v.reshape(H, hd)
    half = hd // 2
    np.testing.assert_allclose(r[:, :half] ** 2 + r[:, half:] ** 2, vv[:, :half] ** 2 + vv[:, half:] ** 2,
                               rtol=1e-5)                                # pair norms preserved
    a = ora.op_rope(ora.op_rope(v, H, hd, 7, base), H, hd, 30, base)    # rotations compose
    np.testing.assert_allclose(a, ora.op_rope(v, H, hd, 37, base), atol=2e-6)
    # closed form: hd=2, theta_0 = 1: (x0, x1) -> (x0 cos p - x1 sin p, x1 cos p + x0 sin p)
    out = ora.op_rope(np.array([2.0, 0.5], np.float32), 1, 2, 3, base)
    np.testing.assert_allclose(out, [2 * math.cos(3) - 0.5 * math.sin(3), 0.5 * math.cos(3) + 2 * math.sin(3)],
                               rtol=1e-6)
    # frequencies: theta_i = base^(-2i/hd); pair i of a unit vector at pos 1 rotates by theta_i
    hd2 = 8
    for i in range(hd2 // 2):
        e = np.zeros(hd2, np.float32)
        e[i] = 1
        o = ora.op_rope(e, 1, hd2, 1, 100.0)
        th = 100.0 ** (-2.0 * i / hd2)
        np.testing.assert_allclose([o[i], o[i + hd2 // 2]], [math.cos(th), math.sin(th)], atol=1e-7)


def test_rope_relative_position_property():
    hd, base = 32, 1e4
    q = rng.standard_normal(hd).astype(np.float32)
    k = rng.standard_normal(hd).astype(np.float32)
    d1 = float(ora.op_rope(q, 1, hd, 50, base) @ ora.op_rope(k, 1, hd, 20, base))
    d2 = float(ora.op_rope(q, 1, hd, 130, base) @ ora.op_rope(k, 1, hd, 100, base))
    assert abs(d1 - d2) < 1e-4


def _attn_ref(q, K, V, Hq, Hkv, hd):
    q = q.reshape(Hq, hd).astype(np.float64)
    K = si.bf16_bits_to_f32(K).astype(np.float64).reshape(-1, Hkv, hd)
    V = si.bf16_bits_to_f32(V).astype(np.float64).reshape(-1, Hkv, hd)
    out = np.zeros((Hq, hd))
    for h in range(Hq):
        kv = h // (Hq // Hkv)
        s = torch.from_numpy(K[:, kv] @ q[h] / math.sqrt(hd))
        w = torch.softmax(s, dim=0).numpy()
        out[h] = w @ V[:, kv]
    return out.reshape(-1)


@pytest.mark.parametrize("Hq,Hkv,hd,T", [(4, 2, 64, 37), (4, 4, 16, 5), (8, 1, 32, 130)])
def test_attention_matches_library_softmax(Hq, Hkv, hd, T):
    q = rng.standard_normal(Hq * hd).astype(np.float32)
    K = bf16(rng.standard_normal((T, Hkv * hd)))
    V = bf16(rng.standard_normal((T, Hkv * hd)))
    np.testing.assert_allclose(ora.op_attention(q, K, V, Hq, Hkv, hd), _attn_ref(q, K, V, Hq, Hkv, hd),
                               rtol=1e-5, atol=1e-6)


def test_attention_special_cases():
    Hq, Hkv, hd = 4, 2, 8
    q = rng.standard_normal(Hq * hd).astype(np.float32)
    V = bf16(rng.standard_normal((6, Hkv * hd)))
    K = bf16(rng.standard_normal((6, Hkv * hd)))
    Vf = si.bf16_bits_to_f32(V).reshape(6, Hkv, hd)
    # T = 1: the output is the single V row exactly, per kv-head group
    o = ora.op_attention(q, K[:1], V[:1], Hq, Hkv, hd).reshape(Hq, hd)
    for h in range(Hq):
        assert np.array_equal(o[h], Vf[0, h // 2])
    # q = 0: uniform weights -> mean of V rows
    o = ora.op_attention(np.zeros_like(q), K, V, Hq, Hkv, hd).reshape(Hq, hd)
    for h in range(Hq):
        np.testing.assert_allclose(o[h], Vf[:, h // 2].mean(axis=0), rtol=1e-6, atol=1e-7)
    # a dominant score selects its row (softmax limit): K row 3 of kv-head 1 = 50*q_h2 direction
    K2 = si.bf16_bits_to_f32(K).reshape(6, Hkv, hd).copy()
    K2[:, 1] = 0
    K2[3, 1] = 60 * q.reshape(Hq, hd)[2] / np.linalg.norm(q.reshape(Hq, hd)[2])
    o = ora.op_attention(q * 10, bf16(K2.reshape(6, -1)), V, Hq, Hkv, hd).reshape(Hq, hd)
    np.testing.assert_allclose(o[2], Vf[3, 1], atol=1e-5)


def test_silu_mul_and_argmax():
    g = np.array([0.0, 1.0, -2.0, 30.0, -30.0], np.float32)
    u = np.array([5.0, 2.0, 3.0, 1.0, 1.0], np.float32)
    want = torch.nn.functional.silu(torch.tensor(g, dtype=torch.float64)).numpy() * u
    np.testing.assert_allclose(ora.op_silu_mul(g, u), want, rtol=1e-6, atol=1e-12)
    assert ora.op_silu_mul(g, u)[0] == 0.0
    assert ora.op_argmax(np.array([1, 5, 5, 2, 5], np.float32)) == 1      # lowest index among ties
    assert ora.op_argmax(np.array([-3, -1, -2], np.float32)) == 1
