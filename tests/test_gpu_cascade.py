"""Multi-level (tree) cascade: probes forked from the main stream at successive
CoT positions (Algorithm 1 steps 4-6; Fig. 4) share nested prefixes.
The oracle ignores groups altogether -- that IS the pin: the result does not depend on how the
planner cuts the sharing -- so every test compares all outputs with it and checks what the plan says
it reads against the nested unique-token model."""
import numpy as np
import pytest

import synth
from _harness import Both, assert_state_equal, check_attn, make_oracle, make_spork

pytestmark = pytest.mark.gpu


def _build(cfg, stride, k_per_seq=None, extra=64):
    wl = synth.SuccessiveWorkload(cfg, stride, k_per_seq)
    per_seq = int(wl.total_len.max()) // 16 + 3
    npg = int(sum(int(x) // 16 + 2 for x in wl.total_len)) + extra
    orc, spk = make_oracle(cfg, npg, cfg.n_seqs + 4, per_seq), make_spork(cfg, npg, cfg.n_seqs + 4, per_seq)
    ids = synth.build_state_successive(Both(orc, spk), wl)
    return wl, orc, spk, ids


@pytest.mark.parametrize("n_probes,stride,prefix", [(2, 512, 4096), (3, 500 + 12, 2048), (6, 256, 1024), (3, 144, 520)])
def test_successive_probes_decode(n_probes, stride, prefix):
    cfg = synth.CFG3.scaled(n_groups=2, group_size=n_probes + 1, prefix_len=prefix, suffix_lo=1, suffix_hi=180)
    wl, orc, spk, ids = _build(cfg, stride)
    assert_state_equal(orc, spk, ids)
    q = wl.q_all()
    ref, lref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, ref, lref, "bf16", f"{n_probes} successive probes")
    info = spk.last_plan()
    assert info["unique_tokens"] == wl.unique_tokens()          # every shared token is read once
    assert info["n_levels"] == n_probes                         # P, P+s, ..., P+(R-1)s are shared; beyond that main is alone
    # one shared level only (the round-1 planner): same result, more reads
    spk.set_cascade_levels(1)
    out1, lse1 = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out1, lse1, ref, lref, "bf16", "single level")
    info1 = spk.last_plan()
    assert info1["n_levels"] == 1
    assert info1["unique_tokens"] == wl.single_level_tokens() > info["unique_tokens"]
    # two levels
    spk.set_cascade_levels(2)
    out2, lse2 = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out2, lse2, ref, lref, "bf16", "two levels")
    assert spk.last_plan()["n_levels"] == min(2, n_probes)
    assert info["unique_tokens"] <= spk.last_plan()["unique_tokens"] <= info1["unique_tokens"]


def test_successive_probes_verify_and_mixed_groups():
    """verify (ragged k) over nested sharing; the members are listed in an order that makes the trie's
    subsets non-contiguous in the call (row map), and one unrelated sequence joins a group."""
    cfg = synth.CFG2.scaled(n_groups=2, group_size=4, prefix_len=1024 + 16, suffix_lo=0, suffix_hi=120)
    ks = np.array([3, 1, 7, 4, 2, 9, 1, 5])
    wl, orc, spk, ids = _build(cfg, 192, ks)
    q, qi = wl.q_all(), wl.q_indptr()
    ref, lref = orc.verify(ids, qi, q)
    out, lse = spk.verify_attn(wl.group_indptr(), ids, qi, q)
    check_attn(out, lse, ref, lref, "bf16", "nested verify")
    assert spk.last_plan()["n_levels"] == 3 and spk.last_plan()["unique_tokens"] == wl.unique_tokens()
    # permuted members: [probe 2, main, probe 1, probe 3] -> {probe 2, main, probe 3} share more than probe 1
    perm = np.array([2, 0, 1, 3, 6, 4, 5, 7])
    ids_p = ids[perm]
    q_rows = [q[qi[i]:qi[i + 1]] for i in range(len(ids))]
    q_p = np.concatenate([q_rows[i] for i in perm], axis=0)
    qi_p = np.concatenate([[0], np.cumsum(ks[perm])]).astype(np.int32)
    ref_p, lref_p = orc.verify(ids_p, qi_p, q_p)
    out_p, lse_p = spk.verify_attn(wl.group_indptr(), ids_p, qi_p, q_p)
    check_attn(out_p, lse_p, ref_p, lref_p, "bf16", "nested verify, permuted members")
    assert spk.last_plan()["unique_tokens"] == wl.unique_tokens()
    # one big declared group of everything: the two fork families share nothing with each other
    ref_a, lref_a = orc.decode(ids, q[qi[:-1]])
    out_a, lse_a = spk.decode_attn([0, len(ids)], ids, q[qi[:-1]])
    check_attn(out_a, lse_a, ref_a, lref_a, "bf16", "two families in one declared group")


def test_fork_of_fork_and_truncate_reappend():
    """Lineage corner cases: a probe forked from a probe; a main stream rolled back below a fork point
    and extended again (its new pages are NOT the pages its children hold at those indices)."""
    cfg = synth.CFG5.scaled(n_groups=1, group_size=1)
    orc, spk = make_oracle(cfg, 600, 12, 120), make_spork(cfg, 600, 12, 120)
    both = Both(orc, spk)
    r = np.random.default_rng(3)

    def tok(n):
        return (synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), "bf16"),
                synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), "bf16"))

    def check(seqs, what):
        seqs = np.asarray(seqs, np.int32)
        q = synth.to_storage(r.standard_normal((len(seqs), cfg.Hq, cfg.D), dtype=np.float32), "bf16")
        ref, lref = orc.decode(seqs, q)
        out, lse = spk.decode_attn([0, len(seqs)], seqs, q)
        check_attn(out, lse, ref, lref, "bf16", what)
        return spk.last_plan()

    main = int(both.seq_create(1)[0])
    both.append([main], [640], *tok(640))
    p1 = int(both.fork([main])[0])
    both.append([p1], [200], *tok(200))
    p2 = int(both.fork([p1])[0])                       # fork of a fork: shares 640 with main, 832 with p1
    both.append([main], [300], *tok(300))
    both.append([p2], [37], *tok(37))
    both.append([p1], [5], *tok(5))
    info = check([main, p1, p2], "fork of a fork")
    assert info["n_levels"] == 2
    assert info["unique_tokens"] == 640 + 300 + (840 // 16) * 16 - 640 + (845 - 832) + (877 - 832)
    assert_state_equal(orc, spk, [main, p1, p2])
    # main rolled back to 400 tokens (below the fork point), then extended past it again
    both.truncate([main], [400])
    both.append([main], [500], *tok(500))
    info = check([main, p1, p2], "after rollback below the fork point")
    assert info["unique_tokens"] == 400 + 500 + (832 - 400) + (845 - 832) + (877 - 832)
    assert_state_equal(orc, spk, [main, p1, p2])
    # release the middle of the chain: p2 keeps its pages, sharing with main is unchanged
    both.release([p1])
    info = check([main, p2], "parent of p2 released")
    assert info["unique_tokens"] == 400 + 500 + (877 - 400)
    both.release([main, p2])
    assert not spk.export_refcounts().any() and spk.status() == 0
