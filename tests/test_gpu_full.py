"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the oracle
holds the SAME state (built through the same call script, K/V stored) and EVERY output element of
every configuration is compared with its plain fp64 definition; block tables, lengths and refcounts
are compared bit for bit."""
import numpy as np
import pytest

import synth
from _harness import Both, assert_state_equal, check_attn, make_oracle, sampled_rows_check

pytestmark = pytest.mark.gpu


def _build_both(cfg, k_per_seq=None):
    import bench
    import paper_2607_03333_b200 as sp
    wl = synth.Workload(cfg, k_per_seq)
    npg, mp = bench.pool_dims(wl)
    orc = make_oracle(cfg, npg, cfg.n_seqs + 8, mp)
    spk = sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, npg, cfg.n_seqs + 8, mp, cfg.scale)
    ids = synth.build_state(Both(orc, spk), wl)
    return wl, orc, spk, ids


def _state_properties(spk, wl, ids):
    c = wl.cfg
    rc = spk.export_refcounts()
    total_pages = 0
    for g in range(c.n_groups):
        mem = wl.members(g)
        tabs = [spk.export(int(ids[m])) for m in mem]
        nshared = c.prefix_len // 16
        for (L, T), m in zip(tabs, mem):
            assert L == int(wl.total_len[m])
            assert np.array_equal(T[:nshared], tabs[0][1][:nshared])      # shared prefix pages
            total_pages += len(T)
        assert np.all(rc[tabs[0][1][:nshared]] == c.group_size)
        priv = np.concatenate([T[nshared:] for _, T in tabs])
        assert len(np.unique(priv)) == len(priv) and np.all(rc[priv] == 1)
    assert int(rc.sum()) == total_pages
    assert spk.free_pages() == int((rc == 0).sum()) and spk.status() == 0


@pytest.mark.parametrize("n", [2, 3, 5])
def test_full_decode_configs_every_row(n):
    cfg = synth.CONFIGS[n]
    wl, orc, spk, ids = _build_both(cfg)
    assert_state_equal(orc, spk, ids)
    _state_properties(spk, wl, ids)
    q = wl.q_all()
    ref, lref = orc.decode(ids, q)                      # the whole step, fp64, plain definition
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    info = spk.last_plan()
    assert info["kernel"] == 2 and info["stream_k"] == 1 and info["unique_tokens"] == wl.unique_tokens()
    assert info["n_prefix_items"] > 0
    check_attn(out, lse, ref, lref, "bf16", f"{cfg.name} (all {ref.shape[0] * ref.shape[1]} rows)")
    # the other schedule of the same kernel, and the mma.sync kernel, at full size
    spk.set_stream_k(False)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    assert spk.last_plan()["stream_k"] == 0
    check_attn(out, lse, ref, lref, "bf16", f"{cfg.name} chunked schedule")
    spk.set_stream_k(True)
    if n == 2:
        spk.set_tensor_path_min_rows(1 << 20)
        out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
        assert spk.last_plan()["kernel"] == 1
        check_attn(out, lse, ref, lref, "bf16", f"{cfg.name} mma.sync kernel")


def test_full_verify_config4_every_row():
    """config 4 at k = 16, then the same state rolled back (spork_truncate, on both sides) to k = 8 and
    k = 4: every output row of each against the oracle."""
    cfg = synth.CFG4.scaled(k_draft=16)
    wl, orc, spk, ids = _build_both(cfg)
    both = Both(orc, spk)
    for k in (16, 8, 4):
        cfgk = synth.CFG4.scaled(k_draft=k)
        wlk = synth.Workload(cfgk)
        if k != 16:
            both.truncate(ids, wlk.total_len.astype(np.int32))
        assert_state_equal(orc, spk, ids)
        q, qi = wlk.q_all(), wlk.q_indptr()
        ref, lref = orc.verify(ids, qi, q)
        for variant in ((0, 1, 2) if k == 16 else (0,)):
            spk.set_many_row_variant(variant)
            out, lse = spk.verify_attn(wlk.group_indptr(), ids, qi, q)
            info = spk.last_plan()
            assert info["unique_tokens"] == wlk.unique_tokens()
            assert (info["n_two_pipe_items"] > 0) == (variant != 0)
            check_attn(out, lse, ref, lref, "bf16", f"cfg4 k={k} variant {variant} (all rows)")
        spk.set_many_row_variant(0)
        if k == 4:
            # a directly built k = 4 state holds the same values (independent sub-streams): sampled rows
            # against the dense definition on regenerated K/V
            sampled_rows_check(out, lse, wlk, [(3, 1, 5), (40, 3, 63)], "cfg4 k=4 regenerated")
    both.release(ids)
    assert not spk.export_refcounts().any() and spk.status() == 0


def test_cfg5_fork_churn_on_1m_page_pool():
    """10,000 forks + releases over a 2^20-page pool: refcounts and free count return exactly."""
    import paper_2607_03333_b200 as sp
    cfg = synth.CFG5.scaled(n_groups=4, prefix_len=32768, suffix_lo=1, suffix_hi=4096)
    wl = synth.Workload(cfg)
    spk = sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, 1 << 20, cfg.n_seqs + 10008,
                   int(wl.total_len.max()) // 16 + 4, cfg.scale)
    ids = synth.build_state(spk, wl)
    rc0 = spk.export_refcounts()
    free0 = spk.free_pages()
    parents = synth.churn_parents(5, 10000, ids)
    ch = spk.fork(parents)
    assert len(np.unique(ch)) == 10000
    rc1 = spk.export_refcounts()
    n_tail = int(sum(int(wl.total_len[list(ids).index(p)]) % 16 != 0 for p in parents))
    assert spk.free_pages() == free0 - n_tail
    # every parent's full pages gained exactly (number of its forks) references
    cnt = np.bincount(parents, minlength=int(ids.max()) + 1)
    for s in ids[:6]:
        L, T = spk.export(int(s))
        nf = L // 16
        own = T[cfg.prefix_len // 16:nf]          # private full pages: 1 + forks of this sequence
        assert np.all(rc1[own] == 1 + cnt[int(s)])
    # children: same length, same full pages, private tail
    for c_, p in list(zip(ch, parents))[:8]:
        Lc, Tc = spk.export(int(c_))
        Lp, Tp = spk.export(int(p))
        assert Lc == Lp and np.array_equal(Tc[:Lc // 16], Tp[:Lp // 16])
        if Lc % 16:
            assert Tc[-1] != Tp[-1] and rc1[Tc[-1]] == 1
    spk.release(ch)
    assert np.array_equal(spk.export_refcounts(), rc0) and spk.free_pages() == free0
    spk.release(ids)
    assert not spk.export_refcounts().any() and spk.free_pages() == (1 << 20) and spk.status() == 0


def test_cfg5_churn_oracle_parity_lengths_only():
    """The churn step against the oracle at config 5's full lengths (values do not matter to the
    allocator: both sides replay the call script with zero K/V): tables of sampled children, every
    refcount, before and after the release."""
    import paper_2607_03333_b200 as sp
    import bench
    cfg = synth.CFG5
    wl = synth.Workload(cfg)
    npg, mp = bench.pool_dims(wl)
    npg += 10100
    orc = make_oracle(cfg, npg, cfg.n_seqs + 10008, mp, store_kv=False)
    spk = sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, npg, cfg.n_seqs + 10008, mp, cfg.scale)
    ids = synth.build_state(Both(orc, spk), wl, values=False)
    parents = synth.churn_parents(5, 10000, ids)
    ch = Both(orc, spk).fork(parents)
    assert_state_equal(orc, spk, list(ids[::17]) + list(ch[::97]))
    Both(orc, spk).release(ch)
    assert_state_equal(orc, spk, ids[::5])
