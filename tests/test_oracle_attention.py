"""Pins for the oracle's attention routines (CPU only).

Each test checks oracle/spork_oracle.c against something OTHER than itself:
closed forms, invariants, an independently written numpy float64 computation on
dense gathers, torch's float64 scaled_dot_product_attention (library special
case), and the six invariants BASELINE.json `north_star` lists.  The paper
prints no worked numeric example for this path, so there
is no paper fixture to compare with; see tests/golden/README.md.
"""
import math

import numpy as np
import pytest
import torch

import oracle
import synth


def mk(dtype="f32", Hq=4, Hkv=2, D=8, num_pages=64, max_seqs=8, mpps=16, scale=None):
    scale = 1.0 / math.sqrt(D) if scale is None else scale
    return oracle.Oracle(dtype, Hq, Hkv, D, num_pages, max_seqs, mpps, scale)


def rand_store(r, shape, dtype):
    return synth.to_storage(r.standard_normal(shape, dtype=np.float32), dtype)


def one_seq(o, L, r, dtype="f32"):
    sid = o.seq_create(1)
    k = rand_store(r, (L, o.Hkv, o.D), dtype)
    v = rand_store(r, (L, o.Hkv, o.D), dtype)
    if L:
        o.append(sid, [L], k, v)
    return int(sid[0]), k, v


def numpy_attention(q, K, V, scale):
    """independent float64 definition: softmax(scale * K q) @ V, natural-log lse"""
    s = scale * (K @ q)
    m = s.max()
    w = np.exp(s - m)
    return (w / w.sum()) @ V, m + math.log(w.sum())


# ---- closed forms --------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_single_key_returns_its_value(dtype):
    r = np.random.default_rng(1)
    o = mk(dtype)
    sid, k, v = one_seq(o, 1, r, dtype)
    q = rand_store(r, (1, o.Hq, o.D), dtype)
    out, lse = o.decode([sid], q)
    kf, vf, qf = (synth.storage_to_f64(x, dtype) for x in (k, v, q))
    for h in range(o.Hq):
        c = h // (o.Hq // o.Hkv)
        np.testing.assert_array_equal(out[0, h], vf[0, c])          # exact: p = 1
        s0 = o.scale * float(np.dot(qf[0, h], kf[0, c]))
        assert abs(lse[0, h] - s0) <= 1e-14 * max(1.0, abs(s0))


def test_identical_keys_return_mean_value():
    r = np.random.default_rng(2)
    o = mk()
    L = 37
    sid = o.seq_create(1)
    k1 = r.standard_normal((1, o.Hkv, o.D)).astype(np.float32)
    k = np.repeat(k1, L, axis=0)
    v = r.standard_normal((L, o.Hkv, o.D)).astype(np.float32)
    o.append(sid, [L], k, v)
    q = r.standard_normal((1, o.Hq, o.D)).astype(np.float32)
    out, lse = o.decode(sid, q)
    for h in range(o.Hq):
        c = h // 2
        np.testing.assert_allclose(out[0, h], v[:, c].astype(np.float64).mean(0), rtol=0, atol=1e-14)
        s = o.scale * float(np.dot(q[0, h].astype(np.float64), k1[0, c].astype(np.float64)))
        assert abs(lse[0, h] - (s + math.log(L))) < 1e-13


def test_zero_query_returns_mean_and_log_len():
    r = np.random.default_rng(3)
    o = mk()
    sid, k, v = one_seq(o, 50, r)
    q = np.zeros((1, o.Hq, o.D), np.float32)
    out, lse = o.decode([sid], q)
    for h in range(o.Hq):
        np.testing.assert_allclose(out[0, h], v[:, h // 2].astype(np.float64).mean(0), atol=1e-14)
        assert abs(lse[0, h] - math.log(50)) < 1e-14


def test_softmax_rows_sum_to_one_and_ones_value():
    r = np.random.default_rng(4)
    o = mk()
    sid, k, v = one_seq(o, 45, r)
    q = (3.0 * r.standard_normal((o.Hq, o.D))).astype(np.float32)
    for h in range(o.Hq):
        _, _, p = o.attend_range(sid, h, q[h], 0, 45, probs=True)
        assert abs(p.sum() - 1.0) < 1e-12 and (p >= 0).all()
    # V = 1 everywhere -> out = sum_t p_t = 1
    o2 = mk()
    sid2 = o2.seq_create(1)
    o2.append(sid2, [45], k, np.ones_like(v))
    out, _ = o2.decode(sid2, q[None])
    np.testing.assert_allclose(out, 1.0, atol=1e-12)


def test_one_hot_limit():
    """scaling one key's score up drives the output to that key's value"""
    r = np.random.default_rng(5)
    o = mk(Hq=2, Hkv=2)
    L = 20
    sid = o.seq_create(1)
    k = r.standard_normal((L, 2, o.D)).astype(np.float32)
    v = r.standard_normal((L, 2, o.D)).astype(np.float32)
    q = r.standard_normal((1, 2, o.D)).astype(np.float32)
    k[7] = 200.0 * q[0] / np.linalg.norm(q[0], axis=-1, keepdims=True)   # huge positive score at t=7
    o.append(sid, [L], k, v)
    out, lse = o.decode(sid, q)
    np.testing.assert_allclose(out[0], v[7].astype(np.float64), atol=1e-12)
    for h in range(2):
        s7 = o.scale * float(np.dot(q[0, h].astype(np.float64), k[7, h].astype(np.float64)))
        assert abs(lse[0, h] - s7) < 1e-9


def test_token_permutation_invariance():
    r = np.random.default_rng(6)
    L = 48
    k = r.standard_normal((L, 2, 8)).astype(np.float32)
    v = r.standard_normal((L, 2, 8)).astype(np.float32)
    q = r.standard_normal((1, 4, 8)).astype(np.float32)
    perm = r.permutation(L)
    res = []
    for kk, vv in ((k, v), (k[perm], v[perm])):
        o = mk()
        sid = o.seq_create(1)
        o.append(sid, [L], kk, vv)
        res.append(o.decode(sid, q))
    np.testing.assert_allclose(res[0][0], res[1][0], atol=1e-13)
    np.testing.assert_allclose(res[0][1], res[1][1], atol=1e-13)


# ---- brute force / library ------------------------------------------------------
@pytest.mark.parametrize("dtype,Hq,Hkv,D,L", [("f32", 4, 2, 8, 1), ("f32", 4, 1, 8, 16),
                                                ("f32", 6, 3, 4, 33), ("bf16", 8, 2, 16, 64),
                                                ("bf16", 4, 4, 8, 47)])
def test_decode_vs_independent_numpy_and_torch_sdpa(dtype, Hq, Hkv, D, L):
    r = np.random.default_rng(100 + L)
    o = mk(dtype, Hq, Hkv, D)
    sid, k, v = one_seq(o, L, r, dtype)
    q = rand_store(r, (1, Hq, D), dtype)
    out, lse = o.decode([sid], q)
    kf, vf, qf = (synth.storage_to_f64(x, dtype) for x in (k, v, q))
    G = Hq // Hkv
    for h in range(Hq):
        eo, el = numpy_attention(qf[0, h], kf[:, h // G], vf[:, h // G], o.scale)
        np.testing.assert_allclose(out[0, h], eo, atol=1e-13)
        assert abs(lse[0, h] - el) < 1e-12
    # library special case: torch float64 SDPA on the dense gather, GQA expanded by hand
    tq = torch.from_numpy(qf).permute(1, 0, 2)[None]                      # [1, Hq, 1, D]
    tk = torch.from_numpy(kf).permute(1, 0, 2).repeat_interleave(G, 0)[None]   # [1, Hq, L, D]
    tv = torch.from_numpy(vf).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, scale=o.scale)
    np.testing.assert_allclose(out[0], ref[0, :, 0].numpy(), atol=1e-12)


def test_gqa_mapping_is_contiguous():
    """A-10: q head h reads kv head h // G -- make kv heads wildly different"""
    r = np.random.default_rng(8)
    o = mk(Hq=6, Hkv=3, D=4)
    L = 9
    sid = o.seq_create(1)
    k = r.standard_normal((L, 3, 4)).astype(np.float32)
    v = np.zeros((L, 3, 4), np.float32)
    for c in range(3):
        v[:, c] = 10.0 * (c + 1)
    o.append(sid, [L], k, v)
    out, _ = o.decode(sid, r.standard_normal((1, 6, 4)).astype(np.float32))
    for h in range(6):
        np.testing.assert_allclose(out[0, h], 10.0 * (h // 2 + 1), atol=1e-12)


def test_paged_walk_matches_dense_routine_and_fragmented_tables():
    """the block-table walk is pinned by fragmenting the pool: interleaved appends of
    several sequences give non-contiguous, non-monotone page runs"""
    r = np.random.default_rng(9)
    o = mk("bf16", 4, 2, 8, num_pages=64, max_seqs=4, mpps=16)
    ids = o.seq_create(3)
    Ls = [70, 33, 52]
    ks = [rand_store(r, (L, 2, 8), "bf16") for L in Ls]
    vs = [rand_store(r, (L, 2, 8), "bf16") for L in Ls]
    done = [0, 0, 0]
    while any(d < L for d, L in zip(done, Ls)):
        for i in (2, 0, 1):
            n = min(5, Ls[i] - done[i])
            if n:
                o.append([ids[i]], [n], ks[i][done[i]:done[i] + n], vs[i][done[i]:done[i] + n])
                done[i] += n
    _, tab = o.export_seq(ids[0])
    assert list(tab) != sorted(tab) or np.any(np.diff(tab) != 1)     # really fragmented
    q = rand_store(r, (3, 4, 8), "bf16")
    out, lse = o.decode(ids, q)
    for i in range(3):
        for h in range(4):
            eo, el = oracle.attend_dense("bf16", o.scale, q[i, h], ks[i][:, h // 2], vs[i][:, h // 2])
            np.testing.assert_allclose(out[i, h], eo, atol=1e-14)
            assert abs(lse[i, h] - el) < 1e-13
            no, nl = numpy_attention(synth.storage_to_f64(q[i, h], "bf16"),
                                     synth.storage_to_f64(ks[i][:, h // 2], "bf16"),
                                     synth.storage_to_f64(vs[i][:, h // 2], "bf16"), o.scale)
            np.testing.assert_allclose(out[i, h], no, atol=1e-13)
            assert abs(lse[i, h] - nl) < 1e-12


def test_empty_sequence():
    o = mk()
    sid = o.seq_create(1)
    out, lse = o.decode(sid, np.ones((1, o.Hq, o.D), np.float32))
    assert np.all(out == 0) and np.all(np.isneginf(lse))


# ---- cascade routine == plain routine (north_star invariant 1) --------------------
def test_cascade_equals_concatenated_for_every_page_aligned_split():
    r = np.random.default_rng(10)
    o = mk("f32", 4, 2, 8, num_pages=64, mpps=16)
    L = 16 * 5 + 7
    sid, k, v = one_seq(o, L, r)
    q = (2.0 * r.standard_normal((1, 4, 8))).astype(np.float32)
    out, lse = o.decode([sid], q)
    for split in list(range(0, L + 1, 16)):
        for h in range(4):
            co, cl = o.cascade_row(sid, h, q[0, h], split)
            np.testing.assert_allclose(co, out[0, h], atol=1e-12)
            assert abs(cl - lse[0, h]) < 1e-12
    # split == len on an aligned sequence: the suffix part is empty
    o2 = mk()
    sid2, _, _ = one_seq(o2, 32, r)
    out2, lse2 = o2.decode([sid2], q)
    co, cl = o2.cascade_row(sid2, 1, q[0, 1], 32)
    np.testing.assert_allclose(co, out2[0, 1], atol=1e-13)
    assert abs(cl - lse2[0, 1]) < 1e-13


def test_merge2_against_direct_formula_and_empty_parts():
    r = np.random.default_rng(11)
    oa, ob = r.standard_normal(8), r.standard_normal(8)
    la, lb = 1.7, -0.4
    out, lse = oracle.merge2(oa, la, ob, lb)
    wa, wb = math.exp(la), math.exp(lb)
    np.testing.assert_allclose(out, (wa * oa + wb * ob) / (wa + wb), atol=1e-14)
    assert abs(lse - math.log(wa + wb)) < 1e-14
    out, lse = oracle.merge2(oa, -math.inf, ob, lb)
    assert np.array_equal(out, ob) and lse == lb
    out, lse = oracle.merge2(oa, la, ob, -math.inf)
    assert np.array_equal(out, oa) and lse == la
    out, lse = oracle.merge2(oa, -math.inf, ob, -math.inf)
    assert np.all(out == 0) and lse == -math.inf and not np.isnan(out).any()


# ---- verify -------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_verify_rows_equal_decode_of_truncated_sequence(dtype):
    """A-13: row j of k sees t <= L-k+j  <=>  plain decode of the first L-k+j+1 tokens"""
    r = np.random.default_rng(12)
    L, ksz = 45, 5
    o = mk(dtype)
    sid, k, v = one_seq(o, L, r, dtype)
    q = rand_store(r, (ksz, o.Hq, o.D), dtype)
    out, lse = o.verify([sid], [0, ksz], q)
    for j in range(ksz):
        o2 = mk(dtype)
        n = L - ksz + j + 1
        s2 = o2.seq_create(1)
        o2.append(s2, [n], k[:n], v[:n])
        eo, el = o2.decode(s2, q[j:j + 1])
        np.testing.assert_array_equal(out[j], eo[0])
        np.testing.assert_array_equal(lse[j], el[0])


def test_verify_k1_is_decode_and_ragged_batch():
    r = np.random.default_rng(13)
    o = mk()
    ids = o.seq_create(3)
    Ls = [20, 35, 9]
    for i, L in zip(ids, Ls):
        o.append([i], [L], r.standard_normal((L, 2, 8)).astype(np.float32),
                 r.standard_normal((L, 2, 8)).astype(np.float32))
    q1 = r.standard_normal((3, 4, 8)).astype(np.float32)
    vo, vl = o.verify(ids, [0, 1, 2, 3], q1)
    do, dl = o.decode(ids, q1)
    np.testing.assert_array_equal(vo, do)
    np.testing.assert_array_equal(vl, dl)
    # ragged k = (3, 1, 4): each block of rows matches a single-sequence call
    qi = [0, 3, 4, 8]
    q = r.standard_normal((8, 4, 8)).astype(np.float32)
    vo, vl = o.verify(ids, qi, q)
    for n, i in enumerate(ids):
        so, sl = o.verify([i], [0, qi[n + 1] - qi[n]], q[qi[n]:qi[n + 1]])
        np.testing.assert_array_equal(vo[qi[n]:qi[n + 1]], so)
        np.testing.assert_array_equal(vl[qi[n]:qi[n + 1]], sl)


def test_verify_vs_torch_sdpa_with_boolean_mask():
    r = np.random.default_rng(14)
    L, ksz, Hq, Hkv, D = 40, 8, 4, 2, 8
    o = mk("f32", Hq, Hkv, D)
    sid, k, v = one_seq(o, L, r)
    q = r.standard_normal((ksz, Hq, D)).astype(np.float32)
    out, lse = o.verify([sid], [0, ksz], q)
    G = Hq // Hkv
    tq = torch.from_numpy(q.astype(np.float64)).permute(1, 0, 2)[None]
    tk = torch.from_numpy(k.astype(np.float64)).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    tv = torch.from_numpy(v.astype(np.float64)).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    mask = torch.zeros(ksz, L, dtype=torch.bool)
    for j in range(ksz):
        mask[j, :L - ksz + j + 1] = True          # bottom-right aligned causal
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, attn_mask=mask, scale=o.scale)
    np.testing.assert_allclose(out, ref[0].permute(1, 0, 2).numpy(), atol=1e-12)
    # last row sees everything; first row does not see the later drafts
    full, _ = o.decode([sid], q[-1:])
    np.testing.assert_array_equal(out[-1], full[0])
    assert np.abs(out[0] - o.decode([sid], q[:1])[0][0]).max() > 1e-6


def test_verify_rejects_bad_k():
    r = np.random.default_rng(15)
    o = mk()
    sid, _, _ = one_seq(o, 3, r)
    rc, _, _ = o.verify([sid], [0, 4], np.zeros((4, 4, 8), np.float32), check=False)
    assert rc == oracle.ERR_INVALID


# ---- fork-related attention invariants (north_star 2) -----------------------------
@pytest.mark.parametrize("L", [32, 39])
def test_fork_with_empty_suffix_equals_parent(L):
    r = np.random.default_rng(16)
    o = mk("bf16")
    sid, k, v = one_seq(o, L, r, "bf16")
    ch = o.fork([sid, sid])
    q = rand_store(r, (1, o.Hq, o.D), "bf16")
    po, pl = o.decode([sid], q)
    for c in ch:
        co, cl = o.decode([c], q)
        np.testing.assert_array_equal(co, po)
        np.testing.assert_array_equal(cl, pl)
    # releasing the parent first leaves the children's attention unchanged
    o.release([sid])
    co, cl = o.decode([ch[0]], q)
    np.testing.assert_array_equal(co, po)
    # and a child's private suffix does not leak into its sibling
    o.append([ch[0]], [3], rand_store(r, (3, 2, 8), "bf16"), rand_store(r, (3, 2, 8), "bf16"))
    so, _ = o.decode([ch[1]], q)
    np.testing.assert_array_equal(so, po)


def test_synth_bf16_rounding_is_rne_and_exact_roundtrip():
    x = np.array([1.0, 1.00390625, 1.0 + 2 ** -8, 1.0 + 3 * 2 ** -8, -2.5, 3.1415927, 1e-30, 65504.0],
                 np.float32)
    bits = synth.f32_to_bf16_bits(x)
    t = torch.from_numpy(x).to(torch.bfloat16)           # library RNE
    np.testing.assert_array_equal(synth.bf16_bits_to_f32(bits), t.to(torch.float32).numpy())
    # ties: 1 + 2^-8 is exactly half way between 1 and 1 + 2^-7 -> even mantissa (1.0)
    assert synth.bf16_bits_to_f32(bits)[2] == 1.0
    assert synth.bf16_bits_to_f32(bits)[3] == np.float32(1.0 + 2 ** -6)
