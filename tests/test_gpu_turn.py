"""The partial-token-accept turn without a host round trip, captured in ONE CUDA graph and replayed
("end-to-end fork -> decode -> verify -> accept -> rollback step under one CUDA
graph"; "in the same decode step"; Algorithm 1 steps 4-5):

    append k_i drafts -> verify attention -> accept + rollback -> append 1 token -> decode attention

Every replay is compared with the oracle running the same turn call by call: verify / decode outputs
within the bf16 tolerances, accept lengths, lengths, block tables and refcounts bit-exact.
"""
import numpy as np
import pytest

import synth
from _harness import assert_state_equal, check_attn, make_oracle, make_spork, pool_dims

pytestmark = pytest.mark.gpu


def _inputs(cfg, ks, turn, accept_upto):
    """seeded inputs of one turn: draft KV, verify q, draft / target tokens, the next token's KV, decode q"""
    r = synth.rng(cfg.cfg_no, synth.T_MISC, 1000 + turn)
    tot, n = int(ks.sum()), len(ks)
    f = lambda *shape: synth.to_storage(r.standard_normal(shape, dtype=np.float32), cfg.dtype)
    fq = lambda *shape: synth.to_storage(r.standard_normal(shape, dtype=np.float32), cfg.q_dtype)
    draft = r.integers(0, 50000, size=tot).astype(np.int32)
    target = draft.copy()
    qi = np.concatenate([[0], np.cumsum(ks)])
    for i in range(n):                       # first mismatch of sequence i at position a_i (a_i = k_i: all accepted)
        a = int(r.integers(0, ks[i] + 1)) if accept_upto is None else min(int(ks[i]), accept_upto)
        if a < ks[i]:
            target[qi[i] + a] += 1
            target[qi[i] + a + 1:qi[i + 1]] = r.integers(0, 50000, size=int(ks[i]) - a - 1)
    return dict(kd=f(tot, cfg.Hkv, cfg.D), vd=f(tot, cfg.Hkv, cfg.D), qv=fq(tot, cfg.Hq, cfg.D), draft=draft,
                target=target, k1=f(n, cfg.Hkv, cfg.D), v1=f(n, cfg.Hkv, cfg.D), qd=fq(n, cfg.Hq, cfg.D))


@pytest.mark.parametrize("ks,n_turns,dtype", [([16, 16, 16, 16], 20, "bf16"), ([4, 9, 16, 1], 20, "bf16"),
                                              ([64, 33, 17, 2], 6, "bf16"), ([8, 3, 16, 5], 8, "e4m3")])
def test_graph_replay_matches_the_oracle_turn_by_turn(ks, n_turns, dtype):
    import torch
    cfg = synth.CFG4.scaled(n_groups=2, prefix_len=1024 + 32, suffix_lo=0, suffix_hi=100, k_draft=0, dtype=dtype)
    wl = synth.Workload(cfg)
    ks = np.array(ks * cfg.n_groups, np.int64)
    grow = int(n_turns * (ks.max() + 1) + ks.max())
    npg, ms, mp = pool_dims(wl, 64 + cfg.n_seqs * (grow // 16 + 2))
    mp += grow // 16 + 2
    orc, spk = make_oracle(cfg, npg, ms, mp), make_spork(cfg, npg, ms, mp)
    ids = synth.build_state(orc, wl)
    assert np.array_equal(ids, synth.build_state(spk, wl))
    gi = wl.group_indptr()
    qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
    tot, n = int(ks.sum()), len(ids)

    dev = spk.device
    st = {k: spk._dev(v) for k, v in _inputs(cfg, ks, 0, None).items()}       # static device buffers
    out_v = torch.empty((tot, cfg.Hq, cfg.D), dtype=torch.float32, device=dev)
    lse_v = torch.empty((tot, cfg.Hq), dtype=torch.float32, device=dev)
    out_d = torch.empty((n, cfg.Hq, cfg.D), dtype=torch.float32, device=dev)
    lse_d = torch.empty((n, cfg.Hq), dtype=torch.float32, device=dev)
    acc = torch.zeros(n, dtype=torch.int32, device=dev)
    turn = spk.turn(gi, ids, qi)

    def enqueue():
        turn.append(0, st["kd"], st["vd"])
        turn.verify(st["qv"], out_v, lse_v)
        turn.accept(st["draft"], st["target"], acc)
        turn.append(1, st["k1"], st["v1"])
        turn.decode(st["qd"], out_d, lse_d)

    def oracle_turn(x):
        orc.append(ids, ks, x["kd"], x["vd"])
        ov = orc.verify(ids, qi, x["qv"])
        _, a = orc.accept(ids, qi, x["draft"], x["target"])
        orc.append(ids, np.ones(n, np.int32), x["k1"], x["v1"])
        return ov, a, orc.decode(ids, x["qd"])

    def check(x, what):
        assert turn.sync() == 0
        (ov, lv), a, (od, ld) = oracle_turn(x)
        assert np.array_equal(acc.cpu().numpy(), a), what
        check_attn(out_v, lse_v, ov, lv, dtype, what + " verify")
        check_attn(out_d, lse_d, od, ld, dtype, what + " decode")
        assert_state_equal(orc, spk, ids)

    # turn 0 eagerly (also the warm-up the capture needs), then the same calls captured once
    x = _inputs(cfg, ks, 0, None)
    enqueue()
    check(x, "eager turn")
    # while a turn is in flight the host-side calls refuse to guess
    turn.append(0, st["kd"], st["vd"])
    import paper_2607_03333_b200 as sp
    assert spk.release([int(ids[0])], check=False) == sp.ERR_STALE
    assert spk.decode_attn(gi, ids, st["qd"], check=False)[0] == sp.ERR_STALE
    turn.accept(st["draft"], st["draft"] + 1, acc)          # nothing accepted: all k drafts rolled back
    assert turn.sync() == 0
    assert_state_equal(orc, spk, ids)                       # append + full rollback = no change

    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=spk.stream):
        enqueue()
    # (capture does not execute: the state is still the oracle's)
    for t in range(1, n_turns + 1):
        # all-accept, none-accept and random turns
        x = _inputs(cfg, ks, t, {1: 0, 2: 64}.get(t))
        with torch.cuda.stream(spk.stream):
            for k, v in x.items():
                st[k].copy_(torch.from_numpy(v), non_blocking=False)
            g.replay()
        check(x, f"replay {t}")
    lens = np.array([orc.export_seq(int(s))[0] for s in ids])
    assert np.all(lens >= wl.total_len + n_turns) and np.any(lens > wl.total_len + n_turns)
    turn.close()
    spk.release(ids)
    orc.release(ids)
    assert not spk.export_refcounts().any() and spk.status() == 0


def test_turn_out_of_pages_changes_nothing_and_is_reported():
    import torch
    import paper_2607_03333_b200 as sp
    cfg = synth.CFG4.scaled(n_groups=1, prefix_len=256, suffix_lo=5, suffix_hi=5, k_draft=0)
    wl = synth.Workload(cfg)
    need = cfg.prefix_len // 16 + cfg.n_seqs           # prefix pages + one private page each: a full pool
    orc, spk = make_oracle(cfg, need, 8, 64), make_spork(cfg, need, 8, 64)
    ids = synth.build_state(orc, wl)
    assert np.array_equal(ids, synth.build_state(spk, wl))
    ks = np.full(cfg.n_seqs, 16, np.int64)              # 5 + 16 tokens need a second private page: none is free
    qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
    x = _inputs(cfg, ks, 0, None)
    turn = spk.turn(wl.group_indptr(), ids, qi)
    turn.append(0, spk._dev(x["kd"]), spk._dev(x["vd"]))
    assert turn.sync(check=False) == sp.ERR_DEVICE
    for s in ids:
        assert spk.export(int(s))[0] == orc.export_seq(int(s))[0]
    assert np.array_equal(spk.export_refcounts(), orc.export_refcounts())
    assert orc.append(ids, ks, x["kd"], x["vd"], check=False) != 0       # the oracle refuses the same append


def test_accept_without_the_turns_drafts_is_refused():
    """spork_turn_accept rolls back drafts the turn appended; asked to roll a sequence back below the length
    the plans were built for, it leaves the sequence alone and reports a device error."""
    import paper_2607_03333_b200 as sp
    cfg = synth.CFG4.scaled(n_groups=1, prefix_len=256, suffix_lo=40, suffix_hi=40, k_draft=0)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 64)
    orc, spk = make_oracle(cfg, npg, ms, mp), make_spork(cfg, npg, ms, mp)
    ids = synth.build_state(orc, wl)
    assert np.array_equal(ids, synth.build_state(spk, wl))
    ks = np.full(cfg.n_seqs, 8, np.int64)
    qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
    x = _inputs(cfg, ks, 0, 0)                        # first mismatch at position 0: every draft rejected
    turn = spk.turn(wl.group_indptr(), ids, qi)
    turn.accept(spk._dev(x["draft"]), spk._dev(x["target"]))     # no drafts were appended by the turn
    assert turn.sync(check=False) == sp.ERR_DEVICE
    assert_lens = [spk.export(int(s))[0] for s in ids]
    assert assert_lens == [orc.export_seq(int(s))[0] for s in ids]
    assert np.array_equal(spk.export_refcounts(), orc.export_refcounts())
