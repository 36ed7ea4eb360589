"""GPU parity of the FP8-KV variant (dtype "e4m3": K and V stored as e4m3 bytes, Q bf16; SURVEY.md 8(f)
NEXT-4, reading B-4) against the fp64 oracle on the same stored bytes.

Tolerances are the bf16 ones (DESIGN.md section 6 derives why): out <= 1e-2, lse 1e-4 relative; block
tables, lengths, refcounts and the stored K/V bytes are bit-exact.  D = 128 runs on the tcgen05 kernel
(e4m3 tiles widened to fp16 in shared memory by the converter warps), other head dims on the CUDA-core
kernel.
"""
import numpy as np
import pytest

import synth
from _harness import assert_state_equal, check_attn, make_oracle, make_spork, pool_dims

pytestmark = pytest.mark.gpu


def _build_both(cfg, k_per_seq=None, extra_pages=64):
    wl = synth.Workload(cfg, k_per_seq)
    npg, ms, mp = pool_dims(wl, extra_pages)
    orc = make_oracle(cfg, npg, ms, mp)
    spk = make_spork(cfg, npg, ms, mp)
    ids_o = synth.build_state(orc, wl)
    ids_s = synth.build_state(spk, wl)
    assert np.array_equal(ids_o, ids_s)
    return wl, orc, spk, ids_o


def f8(cfg, **kw):
    return cfg.scaled(dtype="e4m3", **kw)


SMALL = [
    f8(synth.CFG2, n_groups=3, prefix_len=1000, suffix_lo=1, suffix_hi=300),     # unaligned fork point: tail copies
    f8(synth.CFG3, n_groups=2, prefix_len=1536, suffix_lo=1, suffix_hi=260),     # outlier keys (x8)
    f8(synth.CFG5, n_groups=2, prefix_len=2048 + 16, suffix_lo=1, suffix_hi=200),
    f8(synth.CFG3, n_groups=2, group_size=3, prefix_len=48, suffix_lo=0, suffix_hi=40),
    f8(synth.CFG2, Hq=64, Hkv=4, n_groups=1, group_size=5, prefix_len=640, suffix_lo=0, suffix_hi=90),
]


@pytest.mark.parametrize("stream_k", [True, False])
@pytest.mark.parametrize("cfg", SMALL, ids=lambda c: f"{c.name}-g{c.group_size}-P{c.prefix_len}")
def test_small_e4m3_decode(cfg, stream_k):
    wl, orc, spk, ids = _build_both(cfg)
    spk.set_stream_k(stream_k)
    assert_state_equal(orc, spk, ids)
    # the stored bytes themselves (swizzled 1-byte block image, tail page copies at the fork)
    for s in (ids[0], ids[-1]):
        L = orc.export_seq(int(s))[0]
        ko, vo = orc.read_kv(int(s), 0, L)
        ks, vs = spk.read_kv(int(s), 0, L)
        assert ks.dtype == np.uint8 and np.array_equal(ko, ks) and np.array_equal(vo, vs)
    q = wl.q_all()
    assert q.dtype == np.uint16                       # bf16 queries over an e4m3 cache
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "e4m3", cfg.name)
    info = spk.last_plan()
    assert info["kernel"] == 2 and info["n_umma_items"] == info["n_items"] and info["stream_k"] == int(stream_k)
    if cfg.prefix_len % 16 == 0:                     # (an unaligned fork point keeps its tail tokens private: B-1)
        assert info["unique_tokens"] == wl.unique_tokens()
    # ungrouped (no cascade) gives the same result up to rounding
    out1, lse1 = spk.decode_attn(np.arange(len(ids) + 1), ids, q)
    check_attn(out1, lse1, out_ref, lse_ref, "e4m3", cfg.name + " ungrouped")
    spk.release(ids)
    assert not spk.export_refcounts().any() and spk.status() == 0


@pytest.mark.parametrize("ks", [[4, 8, 16, 1], [16, 16, 16, 16], [3, 7, 12, 5]])
def test_small_e4m3_verify(ks):
    cfg = f8(synth.CFG4, n_groups=2, prefix_len=1024 + 32, suffix_lo=0, suffix_hi=100)
    wl, orc, spk, ids = _build_both(cfg, np.array(ks * cfg.n_groups))
    assert_state_equal(orc, spk, ids)
    q, qi = wl.q_all(), wl.q_indptr()
    out_ref, lse_ref = orc.verify(ids, qi, q)
    out, lse = spk.verify_attn(wl.group_indptr(), ids, qi, q)
    check_attn(out, lse, out_ref, lse_ref, "e4m3", f"verify k={ks}")
    assert spk.last_plan()["kernel"] == 2


def test_e4m3_generic_head_dims_run_on_the_cuda_core_kernel():
    for D, Hq, Hkv in ((64, 8, 2), (96, 6, 3), (256, 4, 1)):
        cfg = f8(synth.CFG2, Hq=Hq, Hkv=Hkv, D=D, n_groups=2, prefix_len=200, suffix_lo=0, suffix_hi=70)
        wl, orc, spk, ids = _build_both(cfg)
        assert_state_equal(orc, spk, ids)
        L = orc.export_seq(int(ids[1]))[0]
        assert np.array_equal(orc.read_kv(int(ids[1]), 0, L)[0], spk.read_kv(int(ids[1]), 0, L)[0])
        q = wl.q_all()
        out_ref, lse_ref = orc.decode(ids, q)
        out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
        check_attn(out, lse, out_ref, lse_ref, "e4m3", f"D={D}")
        assert spk.last_plan()["kernel"] == 0


def test_e4m3_degenerate_cases():
    cfg = f8(synth.CFG2, n_groups=2, prefix_len=256, suffix_lo=0, suffix_hi=0)      # empty suffixes
    wl, orc, spk, ids = _build_both(cfg)
    q = wl.q_all()
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "e4m3", "empty suffix")
    # an empty sequence: out = 0, lse = -inf; one token: out = V exactly (every e4m3 value is an fp32 value)
    e_o, e_s = orc.seq_create(2), spk.seq_create(2)
    r = synth.rng(2, synth.T_MISC, 1)
    k1 = synth.to_storage(r.standard_normal((1, cfg.Hkv, cfg.D), dtype=np.float32), "e4m3")
    v1 = synth.to_storage(r.standard_normal((1, cfg.Hkv, cfg.D), dtype=np.float32), "e4m3")
    orc.append(e_o[1:], [1], k1, v1)
    spk.append(e_s[1:], [1], k1, v1)
    o, l = spk.decode_attn([0, 1, 2], e_s, q[:2])
    o, l = o.cpu().numpy(), l.cpu().numpy()
    assert not o[0].any() and np.all(np.isneginf(l[0]))
    vf = synth.e4m3_bits_to_f32(v1)[0]
    for h in range(cfg.Hq):
        assert np.array_equal(o[1, h], vf[h // cfg.G])
    # subnormal and extreme stored values survive the in-kernel widening: K = V = each finite code once
    codes = np.array([c for c in range(256) if c not in (0x7F, 0xFF)], np.uint8)
    n = 256
    kk = np.resize(codes, (n, cfg.Hkv, cfg.D)).astype(np.uint8)
    vv = np.ascontiguousarray(kk[::-1])
    so, ss = orc.seq_create(1), spk.seq_create(1)
    orc.append(so, [n], kk, vv)
    spk.append(ss, [n], kk, vv)
    qz = synth.to_storage((r.standard_normal((1, cfg.Hq, cfg.D)) * 0.01).astype(np.float32), "bf16")
    o_ref, l_ref = orc.decode(so, qz)
    o, l = spk.decode_attn([0, 1], ss, qz)
    got, want = o.cpu().numpy().astype(np.float64), o_ref
    assert np.max(np.abs(got - want) / np.maximum(1.0, np.abs(want))) <= 1e-2      # values up to 448
    assert np.allclose(l.cpu().numpy(), l_ref, rtol=1e-4, atol=1e-4)


def test_full_config2_shape_in_e4m3_every_row():
    """BASELINE.json config 2's batch with an e4m3 cache: the whole step against the oracle."""
    cfg = f8(synth.CFG2)
    wl, orc, spk, ids = _build_both(cfg)
    assert_state_equal(orc, spk, ids)
    q = wl.q_all()
    ref, lref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    info = spk.last_plan()
    assert info["kernel"] == 2 and info["stream_k"] == 1 and info["unique_tokens"] == wl.unique_tokens()
    check_attn(out, lse, ref, lref, "e4m3", "cfg2 shape, e4m3 KV (all rows)")


def test_full_config5_shape_in_e4m3_every_row():
    """BASELINE.json config 5's batch (128 sequences, prefix 32768) with an e4m3 cache: the whole step against the
    oracle, and the 36-layer-style chained call on two layers of it."""
    import torch
    cfg = f8(synth.CFG5)
    wl, orc, spk, ids = _build_both(cfg)
    assert_state_equal(orc, spk, ids)
    q = wl.q_all()
    ref, lref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    info = spk.last_plan()
    assert info["kernel"] == 2 and info["stream_k"] == 1 and info["unique_tokens"] == wl.unique_tokens()
    check_attn(out, lse, ref, lref, "e4m3", "cfg5 shape, e4m3 KV (all rows)")
    # two layers over the same tables (layer 1 = a copy of layer 0's pools): one plan, chained launches
    spk.layers(2)
    with torch.cuda.stream(spk.stream):
        spk.k_pools[1].copy_(spk.k_pool)
        spk.v_pools[1].copy_(spk.v_pool)
    qd = spk._dev(q)
    outs = [torch.empty_like(out) for _ in range(2)]
    lses = [torch.empty_like(lse) for _ in range(2)]
    spk.attn_layers(wl.group_indptr(), ids, [qd, qd], outs, lses)
    for l in range(2):
        check_attn(outs[l], lses[l], ref, lref, "e4m3", f"cfg5 e4m3, layer {l} of a chained call")
