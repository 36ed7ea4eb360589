"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times:
sampled output rows are compared one by one with the oracle's plain dense definition on
regenerated K/V; block-table / refcount properties that hold at any size are checked too."""
import numpy as np
import pytest

import synth
from _harness import sampled_rows_check

pytestmark = pytest.mark.gpu


def _build(cfg, k_per_seq=None):
    import bench
    wl = synth.Workload(cfg, k_per_seq)
    spk, ids = bench.build_spork(cfg, wl)
    return wl, spk, ids


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


def _samples(wl, n, seed):
    r = np.random.default_rng([11, seed])
    c = wl.cfg
    out = []
    for _ in range(n):
        s = int(r.integers(0, c.n_seqs))
        k = int(wl.k[s])
        out.append((s, int(r.integers(0, max(1, k))), int(r.integers(0, c.Hq))))
    return sorted(out)


@pytest.mark.parametrize("n", [2, 3, 5])
def test_full_decode_configs(n):
    cfg = synth.CONFIGS[n]
    wl, spk, ids = _build(cfg)
    _state_properties(spk, wl, ids)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, wl.q_all())
    info = spk.last_plan()
    assert info["kernel"] in (1, 2, 3) and info["unique_tokens"] == wl.unique_tokens()
    assert info["n_prefix_items"] > 0
    sampled_rows_check(out, lse, wl, _samples(wl, 6, n), cfg.name)
    assert np.all(np.isfinite(out.cpu().numpy()))


@pytest.mark.parametrize("k", [4, 8, 16])
def test_full_verify_config4(k):
    cfg = synth.CFG4.scaled(k_draft=k)
    wl, spk, ids = _build(cfg)
    _state_properties(spk, wl, ids)
    out, lse = spk.verify_attn(wl.group_indptr(), ids, wl.q_indptr(), wl.q_all())
    assert spk.last_plan()["unique_tokens"] == wl.unique_tokens()
    sampled_rows_check(out, lse, wl, _samples(wl, 5, 40 + k), f"cfg4 k={k}")
    assert np.all(np.isfinite(out.cpu().numpy()))


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
