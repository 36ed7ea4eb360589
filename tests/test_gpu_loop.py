"""The paper's decode loop through the C ABI (Algorithm 1 step 5; SURVEY 8(b) call order
"repeat {append 1 token to each live stream; decode_attn}"): the plan built for the first step keeps
serving while the sequences grow (its open-ended items follow the device lengths), and EVERY step's
output is compared with the oracle."""
import numpy as np
import pytest

import synth
from _harness import Both, assert_state_equal, check_attn, make_oracle, make_spork, pool_dims

pytestmark = pytest.mark.gpu


def _tok(r, n, cfg):
    k = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
    v = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
    return k, v


@pytest.mark.parametrize("path", ["tcgen05", "tcgen05-chunked", "mma.sync", "fp32"])
def test_append_one_token_70_steps(path):
    if path == "fp32":
        cfg = synth.CFG1.scaled(n_groups=2, prefix_len=100, suffix_lo=0, suffix_hi=40)
    else:
        cfg = synth.CFG2.scaled(n_groups=3, prefix_len=1000, suffix_lo=1, suffix_hi=300)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 64 + 8 * cfg.n_seqs)
    orc, spk = make_oracle(cfg, npg, ms, mp + 8), make_spork(cfg, npg, ms, mp + 8)
    if path == "mma.sync":
        spk.set_tensor_path_min_rows(1 << 20)
    if path == "tcgen05-chunked":
        spk.set_stream_k(False)
    both = Both(orc, spk)
    ids = synth.build_state(both, wl)
    gi = wl.group_indptr()
    r = np.random.default_rng(5)
    ones = np.ones(cfg.n_seqs, np.int32)
    builds0 = None
    cached = []
    for step in range(70):
        k, v = _tok(r, cfg.n_seqs, cfg)
        both.append(ids, ones, k, v)
        q = synth.to_storage(r.standard_normal((cfg.n_seqs, cfg.Hq, cfg.D), dtype=np.float32), cfg.dtype)
        ref, lref = orc.decode(ids, q)
        out, lse = spk.decode_attn(gi, ids, q)
        check_attn(out, lse, ref, lref, cfg.dtype, f"{path} step {step}")
        info = spk.last_plan()
        cached.append(info["plan_cached"])
        if builds0 is None:
            builds0 = info["plan_builds"]
        assert info["unique_tokens"] == wl.unique_tokens() + (step + 1) * cfg.n_seqs + \
            cfg.n_groups * (cfg.group_size - 1) * (cfg.prefix_len % 16)
    assert_state_equal(orc, spk, ids)
    # one build at the first step, one more when the sequences have grown by a 64-token tile
    assert spk.last_plan()["plan_builds"] - builds0 == 1
    assert sum(cached) == 68 and cached[0] == 0 and cached[64] == 0


def test_verify_loop_appends_drafts_then_rolls_back():
    """k drafts appended -> verify -> accept / rollback -> next turn, several turns: the lengths move
    up and down, the plan is rebuilt after each rollback, every verify output matches the oracle."""
    cfg = synth.CFG4.scaled(n_groups=2, prefix_len=800, suffix_lo=0, suffix_hi=90, k_draft=0)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 256)
    orc, spk = make_oracle(cfg, npg, ms, mp + 8), make_spork(cfg, npg, ms, mp + 8)
    both = Both(orc, spk)
    ids = synth.build_state(both, wl)
    gi = wl.group_indptr()
    r = np.random.default_rng(9)
    for turn in range(6):
        ks = r.integers(1, 13, size=cfg.n_seqs).astype(np.int32)
        qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
        k, v = _tok(r, int(qi[-1]), cfg)
        both.append(ids, ks, k, v)
        q = synth.to_storage(r.standard_normal((int(qi[-1]), cfg.Hq, cfg.D), dtype=np.float32), cfg.dtype)
        ref, lref = orc.verify(ids, qi, q)
        out, lse = spk.verify_attn(gi, ids, qi, q)
        check_attn(out, lse, ref, lref, "bf16", f"turn {turn} verify")
        # the same plan serves a second verify after one more appended token per stream IF k is
        # unchanged: here the drafts differ per turn, so only check the rollback
        d = r.integers(0, 100, size=int(qi[-1])).astype(np.int32)
        t = d.copy()
        for i in range(cfg.n_seqs):
            if r.random() < 0.7:
                t[qi[i] + r.integers(0, ks[i])] += 1
        (rc_o, acc_o), (rc_s, acc_s) = orc.accept(ids, qi, d, t), spk.accept(ids, qi, d, t)
        assert rc_o == rc_s == 0 and np.array_equal(acc_o, acc_s)
        assert_state_equal(orc, spk, ids)
        q1 = synth.to_storage(r.standard_normal((cfg.n_seqs, cfg.Hq, cfg.D), dtype=np.float32), cfg.dtype)
        ref, lref = orc.decode(ids, q1)
        out, lse = spk.decode_attn(gi, ids, q1)
        check_attn(out, lse, ref, lref, "bf16", f"turn {turn} decode after rollback")


def test_verify_plan_follows_growth_with_same_k():
    """verify with the same k after every stream grew: the cached plan's causal limits follow the
    device lengths (ITEM_LEN_LIM)."""
    cfg = synth.CFG4.scaled(n_groups=2, prefix_len=512, suffix_lo=3, suffix_hi=70, k_draft=5)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 128)
    orc, spk = make_oracle(cfg, npg, ms, mp + 8), make_spork(cfg, npg, ms, mp + 8)
    both = Both(orc, spk)
    ids = synth.build_state(both, wl)
    gi, qi = wl.group_indptr(), wl.q_indptr()
    r = np.random.default_rng(12)
    for step in range(20):
        q = synth.to_storage(r.standard_normal((int(qi[-1]), cfg.Hq, cfg.D), dtype=np.float32), cfg.dtype)
        ref, lref = orc.verify(ids, qi, q)
        out, lse = spk.verify_attn(gi, ids, qi, q)
        check_attn(out, lse, ref, lref, "bf16", f"verify step {step}")
        assert spk.last_plan()["plan_cached"] == (1 if step else 0)
        n = r.integers(0, 4, size=cfg.n_seqs).astype(np.int32)
        n[0] = 0                                    # one stream does not grow at all
        k, v = _tok(r, int(n.sum()), cfg)
        both.append(ids, n, k, v)
