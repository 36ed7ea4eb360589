"""Pins of the FP8-KV variant of the oracle (reading B-4): K and V are
stored as e4m3 bytes, Q is bf16; the plain definition is applied to the exactly widened values.

What is pinned here, against things other than the oracle itself:
  * the widening of all 256 e4m3 codes  -> torch.float8_e4m3fn -> float64 (a library's decoder), and the
    format's closed forms (largest finite 448, smallest subnormal 2^-9, +-0, the two NaN codes);
  * the input generator's rounding (synth.f32_to_e4m3_bits) -> torch's round-to-nearest-even cast, and
    round trip / monotonicity / tie-to-even on hand-made cases;
  * attention over e4m3 K/V  -> the same oracle routine fed the SAME values stored as bf16 (every e4m3
    value is exactly representable in bf16, so the two must agree to the last bit), a 5-line numpy
    softmax on the widened values, and torch float64 SDPA;
  * the paged walk with 1-byte elements -> the dense routine; fork tail copy / release invariants on
    an e4m3 pool.
"""
import numpy as np
import pytest
import torch

import oracle
import synth

ALL = np.arange(256, dtype=np.uint8)


def test_widening_of_all_codes_matches_torch_float8():
    want = torch.from_numpy(ALL.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    got = oracle.widen("e4m3", ALL)
    assert np.array_equal(np.isnan(got), np.isnan(want))
    ok = ~np.isnan(want)
    assert np.array_equal(got[ok], want[ok])
    assert np.array_equal(np.signbit(got[ok]), np.signbit(want[ok]))      # -0 keeps its sign
    # the generator's decoder (test-side, independent of the oracle's) agrees as well
    mine = synth.e4m3_bits_to_f32(ALL).astype(np.float64)
    assert np.array_equal(mine[ok], want[ok])


def test_format_closed_forms():
    w = oracle.widen("e4m3", ALL)
    assert w[0x7E] == 448.0 and w[0xFE] == -448.0          # largest finite: 2^8 * 1.75
    assert w[0x01] == 2.0 ** -9 and w[0x07] == 7 * 2.0 ** -9   # subnormals: m/8 * 2^-6
    assert w[0x08] == 2.0 ** -6                            # smallest normal
    assert w[0x38] == 1.0 and w[0x3C] == 1.5 and w[0x40] == 2.0
    assert w[0x00] == 0.0 and w[0x80] == 0.0 and np.signbit(w[0x80])
    assert np.isnan(w[0x7F]) and np.isnan(w[0xFF])
    fin = w[:0x7F]
    assert np.all(np.diff(fin) > 0)                        # codes 0 .. 0x7e are strictly increasing


def test_generator_rounding_matches_torch_and_ties_to_even():
    r = np.random.default_rng(5)
    x = np.concatenate([r.standard_normal(20000) * 8, r.standard_normal(5000) * 0.02,
                        r.uniform(-448, 448, 5000), [0.0, -0.0, 448.0, -448.0, 2.0 ** -9, 2.0 ** -10]]).astype(np.float32)
    got = synth.f32_to_e4m3_bits(x)
    want = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(got, want)
    # every finite code is a fixed point
    codes = np.array([c for c in range(256) if c not in (0x7F, 0xFF)], np.uint8)
    assert np.array_equal(synth.f32_to_e4m3_bits(synth.e4m3_bits_to_f32(codes)), codes)
    # ties go to the even mantissa: 1.0625 -> 1.0 (m=0), 1.1875 -> 1.25 (m=2); 2^-10 -> 0; saturation
    t = synth.e4m3_bits_to_f32(synth.f32_to_e4m3_bits(np.array([1.0625, 1.1875, 2.0 ** -10, 3 * 2.0 ** -10, 1e6, -1e6],
                                                               np.float32)))
    assert list(t) == [1.0, 1.25, 0.0, 2.0 ** -8, 448.0, -448.0]


def _state(seed=0, L=77, Hq=4, Hkv=2, D=32):
    r = np.random.default_rng(seed)
    k8 = synth.f32_to_e4m3_bits((r.standard_normal((L, Hkv, D)) * 2).astype(np.float32))
    v8 = synth.f32_to_e4m3_bits(r.standard_normal((L, Hkv, D)).astype(np.float32))
    q = synth.f32_to_bf16_bits(r.standard_normal((1, Hq, D)).astype(np.float32))
    return k8, v8, q


def test_attention_equals_the_bf16_oracle_on_the_same_values():
    """e4m3 values are a subset of bf16: storing the same numbers as bf16 must change nothing."""
    k8, v8, q = _state()
    L, Hkv, D = k8.shape
    Hq, scale = q.shape[1], 0.2
    k16 = synth.f32_to_bf16_bits(synth.e4m3_bits_to_f32(k8))
    v16 = synth.f32_to_bf16_bits(synth.e4m3_bits_to_f32(v8))
    assert np.array_equal(synth.bf16_bits_to_f32(k16), synth.e4m3_bits_to_f32(k8))     # exact embedding
    outs = []
    for dt, k, v in (("e4m3", k8, v8), ("bf16", k16, v16)):
        o = oracle.Oracle(dt, Hq, Hkv, D, 16, 2, 8, scale)
        s = o.seq_create(1)
        o.append(s, [L], k, v)
        outs.append(o.decode(s, q))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_attention_against_numpy_and_torch_on_widened_values():
    k8, v8, q = _state(seed=3, L=130)
    L, Hkv, D = k8.shape
    Hq, scale = q.shape[1], 1 / np.sqrt(D)
    o = oracle.Oracle("e4m3", Hq, Hkv, D, 16, 2, 10, scale)
    s = o.seq_create(1)
    o.append(s, [L], k8, v8)
    out, lse = o.decode(s, q)
    K = torch.from_numpy(k8.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()   # torch's decoder
    V = torch.from_numpy(v8.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    Q = synth.bf16_bits_to_f32(q).astype(np.float64)
    G = Hq // Hkv
    for h in range(Hq):
        sc = scale * (K[:, h // G] @ Q[0, h])
        w = np.exp(sc - sc.max())
        assert np.allclose(out[0, h], (w / w.sum()) @ V[:, h // G], rtol=0, atol=1e-13)
        assert abs(lse[0, h] - (sc.max() + np.log(w.sum()))) < 1e-12
        ref = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(Q[0, h]).view(1, 1, 1, D), torch.from_numpy(K[:, h // G]).view(1, 1, L, D),
            torch.from_numpy(V[:, h // G]).view(1, 1, L, D), scale=scale)
        assert np.allclose(out[0, h], ref.view(D).numpy(), rtol=0, atol=1e-12)
        # the dense (unpaged) routine on the same bytes
        od, ld = oracle.attend_dense("e4m3", scale, q[0, h], k8[:, h // G], v8[:, h // G])
        assert np.allclose(od, out[0, h], atol=1e-14) and abs(ld - lse[0, h]) < 1e-13


def test_fork_tail_copy_and_release_on_an_e4m3_pool():
    k8, v8, q = _state(seed=9, L=45)       # 45 = 2 full pages + 13 tokens: the fork duplicates a tail page
    L, Hkv, D = k8.shape
    o = oracle.Oracle("e4m3", q.shape[1], Hkv, D, 12, 4, 6, 0.3)
    s = o.seq_create(1)
    o.append(s, [L], k8, v8)
    ch = o.fork(s)
    (Lp, Tp), (Lc, Tc) = o.export_seq(int(s[0])), o.export_seq(int(ch[0]))
    assert Lp == Lc == L and np.array_equal(Tp[:2], Tc[:2]) and Tp[2] != Tc[2]
    kc, vc = o.read_kv(int(ch[0]), 0, L)
    assert np.array_equal(kc, k8) and np.array_equal(vc, v8)          # byte-exact, incl. the copied tail
    a, b = o.decode(s, q), o.decode(ch, q)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])  # empty-suffix child == parent
    o.release(np.concatenate([s, ch]))
    assert not o.export_refcounts().any()


def test_nan_code_is_not_silently_dropped():
    k8, v8, q = _state(seed=1, L=20)
    v8[3, 0, 5] = 0x7F
    o = oracle.Oracle("e4m3", q.shape[1], k8.shape[1], k8.shape[2], 8, 2, 4, 0.2)
    s = o.seq_create(1)
    o.append(s, [20], k8, v8)
    out, _ = o.decode(s, q)
    assert np.isnan(out[0, 0, 5]) and np.isnan(out[0, 1, 5]) and not np.isnan(out[0, 2]).any()
