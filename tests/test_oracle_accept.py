"""Pins of the oracle's partial-token accept (section 4.3: "the first k matching
tokens are accepted") against what the definition fixes: closed forms, an
independently written formulation, and the state invariants of the rollback."""
import numpy as np

import oracle
import synth


def test_accept_len_closed_forms():
    qi = np.array([0, 4, 4 + 8, 4 + 8 + 16, 4 + 8 + 16 + 1])
    d = np.arange(29) % 7
    assert np.array_equal(oracle.accept_len(qi, d, d), [4, 8, 16, 1])          # all match -> k
    t = d.copy()
    t[qi[:-1]] += 1                                                             # first position differs -> 0
    assert np.array_equal(oracle.accept_len(qi, d, t), [0, 0, 0, 0])
    t = d.copy()
    t[[2, 4 + 5, 4 + 8 + 15]] += 3                                              # first mismatch at j -> j
    assert np.array_equal(oracle.accept_len(qi, d, t), [2, 5, 15, 1])
    t[[3, 4 + 7]] += 1                                                          # later mismatches change nothing
    assert np.array_equal(oracle.accept_len(qi, d, t), [2, 5, 15, 1])
    t = d.copy()
    t[1] += 1
    t[0] += 0                                                                   # a match AFTER a mismatch is not counted
    assert oracle.accept_len(qi, d, t)[0] == 1
    assert len(oracle.accept_len(np.array([0]), [], [])) == 0                   # empty batch


def test_accept_len_matches_cumprod_formulation():
    r = np.random.default_rng(5)
    for _ in range(50):
        k = r.integers(1, 20, size=r.integers(1, 9))
        qi = np.concatenate([[0], np.cumsum(k)])
        d = r.integers(0, 3, size=qi[-1])
        t = r.integers(0, 3, size=qi[-1])
        want = [int(np.cumprod(d[a:b] == t[a:b]).sum()) for a, b in zip(qi[:-1], qi[1:])]
        assert np.array_equal(oracle.accept_len(qi, d, t), want)


def test_accept_rolls_back_rejected_drafts():
    cfg = synth.CFG1
    orc = oracle.Oracle(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, 64, 4, 32, cfg.scale)
    r = np.random.default_rng(9)
    ids = orc.seq_create(2)
    lens = [37, 50]
    for s, n in zip(ids, lens):
        kv = r.standard_normal((2, n, cfg.Hkv, cfg.D)).astype(np.float32)
        orc.append([s], [n], kv[0], kv[1])
    ks = [9, 5]                         # the last k tokens of each sequence are drafts
    qi = np.array([0, 9, 14])
    d = np.arange(14)
    t = d.copy()
    t[4] += 1                           # seq 0 accepts 4 of 9; seq 1 accepts all 5
    before = [orc.read_kv(int(s), 0, n) for s, n in zip(ids, lens)]
    rc, acc = orc.accept(ids, qi, d, t)
    assert rc == 0 and np.array_equal(acc, [4, 5])
    new_lens = [37 - (9 - 4), 50]
    for s, n, (k0, v0) in zip(ids, new_lens, before):
        L, T = orc.export_seq(int(s))
        assert L == n and len(T) == (n + 15) // 16
        k1, v1 = orc.read_kv(int(s), 0, n)
        assert np.array_equal(k1, k0[:n]) and np.array_equal(v1, v0[:n])      # the kept prefix is untouched
    rcnt = orc.export_refcounts()
    assert int(rcnt.sum()) == sum((n + 15) // 16 for n in new_lens)             # a whole rejected page is freed
    orc.release(ids)
    assert not orc.export_refcounts().any()
