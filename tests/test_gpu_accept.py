"""GPU parity of the partial-token accept step (spork_accept) and of one whole paper turn
(Algorithm 1, PAPER.md:253-277 + section 4.3): prefill -> fork -> decode -> drafts appended ->
verify -> accept / rollback -> decode again -> release.  Integers are bit-exact."""
import numpy as np
import pytest

import synth
from _harness import assert_state_equal, check_attn, make_oracle, make_spork

pytestmark = pytest.mark.gpu


def _kv(r, n, cfg):
    k = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
    v = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
    return k, v


def _q(r, n, cfg):
    return synth.to_storage(r.standard_normal((n, cfg.Hq, cfg.D), dtype=np.float32), cfg.dtype)


@pytest.mark.parametrize("ks", [[5, 1, 17, 8], [33, 33, 2, 64]])
def test_accept_len_and_rollback(ks):
    cfg = synth.CFG3.scaled(n_groups=1)
    orc, spk = make_oracle(cfg, 256, 8, 64), make_spork(cfg, 256, 8, 64)
    r = np.random.default_rng([3, sum(ks)])
    ids_o, ids_s = orc.seq_create(4), spk.seq_create(4)
    assert np.array_equal(ids_o, ids_s)
    for s, k in zip(ids_s, ks):
        n = 100 + 7 * int(s) + k
        kk, vv = _kv(r, n, cfg)
        orc.append([s], [n], kk, vv)
        spk.append([s], [n], kk, vv)
    qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
    d = r.integers(0, 1000, size=qi[-1]).astype(np.int32)
    t = d.copy()
    # sequence 0: mismatch in the middle, 1: full accept, 2: first token rejected, 3: two mismatches
    t[qi[0] + ks[0] // 2] += 1
    t[qi[2]] += 1
    t[qi[3] + ks[3] - 1] += 1
    t[qi[3] + ks[3] // 3] += 1
    rc_o, acc_o = orc.accept(ids_o, qi, d, t)
    rc_s, acc_s = spk.accept(ids_s, qi, d, t)
    assert rc_o == rc_s == 0
    assert np.array_equal(acc_o, acc_s) and np.array_equal(acc_s, [ks[0] // 2, ks[1], 0, ks[3] // 3])
    assert_state_equal(orc, spk, ids_s)
    # bad arguments change nothing
    import paper_2607_03333_b200 as sp
    bad = qi.copy()
    bad[1:] += 100000
    rc, _ = spk.accept(ids_s, bad, np.zeros(int(bad[-1]), np.int32), np.zeros(int(bad[-1]), np.int32), check=False)
    assert rc == sp.ERR_INVALID
    assert_state_equal(orc, spk, ids_s)
    orc.release(ids_o)
    spk.release(ids_s)
    assert not spk.export_refcounts().any()


def test_one_paper_turn():
    """main prefilled, two probes forked at different CoT positions (Alg. 1 :260-262), everybody
    decodes, a probe is released, main gets k drafts, verify, accept, rollback, decode again."""
    cfg = synth.CFG2.scaled(n_groups=1)
    orc, spk = make_oracle(cfg, 512, 8, 128), make_spork(cfg, 512, 8, 128)
    r = np.random.default_rng(17)
    both = (orc, spk)
    main = int(orc.seq_create(1)[0])
    assert int(spk.seq_create(1)[0]) == main
    kk, vv = _kv(r, 700 + 1, cfg)                       # prefill + first token
    for x in both:
        x.append([main], [701], kk, vv)
    probes = []
    for step in range(2):                               # r * s further CoT tokens, then fork
        kk, vv = _kv(r, 45, cfg)
        for x in both:
            x.append([main], [45], kk, vv)
        po, ps = orc.fork([main]), spk.fork([main])
        assert np.array_equal(po, ps)
        probes.append(int(ps[0]))
        kk, vv = _kv(r, 6, cfg)                         # forced tool-call prefix of the probe
        for x in both:
            x.append([probes[-1]], [6], kk, vv)
    seqs = np.array([main] + probes, np.int32)
    for _ in range(3):                                  # three decode steps of the whole group
        kk, vv = _kv(r, 3, cfg)
        for x in both:
            x.append(seqs, [1, 1, 1], kk, vv)
        q = _q(r, 3, cfg)
        ref, lref = orc.decode(seqs, q)
        out, lse = spk.decode_attn([0, 3], seqs, q)
        check_attn(out, lse, ref, lref, "bf16", "turn decode")
    assert spk.last_plan()["n_prefix_items"] >= 1       # the group shares main's prefix
    assert_state_equal(orc, spk, seqs)
    for x in both:                                      # first probe rejected by the gate / superseded
        x.release([probes[0]])
    k = 12                                              # second probe's body becomes main's drafts (D3)
    kk, vv = _kv(r, k, cfg)
    for x in both:
        x.append([main], [k], kk, vv)
    qi = np.array([0, k], np.int32)
    q = _q(r, k, cfg)
    ref, lref = orc.verify([main], qi, q)
    out, lse = spk.verify_attn([0, 1], [main], qi, q)
    check_attn(out, lse, ref, lref, "bf16", "turn verify")
    d = r.integers(0, 50000, size=k).astype(np.int32)
    t = d.copy()
    t[7] += 1                                           # main's greedy tokens diverge at draft 7
    (rc_o, acc_o), (rc_s, acc_s) = orc.accept([main], qi, d, t), spk.accept([main], qi, d, t)
    assert rc_o == rc_s == 0 and acc_o[0] == acc_s[0] == 7
    live = np.array([main, probes[1]], np.int32)
    assert_state_equal(orc, spk, live)
    q = _q(r, 2, cfg)
    ref, lref = orc.decode(live, q)
    out, lse = spk.decode_attn([0, 2], live, q)
    check_attn(out, lse, ref, lref, "bf16", "decode after rollback")
    for x in both:
        x.release(live)
    assert not spk.export_refcounts().any() and not orc.export_refcounts().any()
    assert spk.status() == 0
