"""GPU parity: libspork (through the C ABI) vs the CPU fp64 oracle, element by
element on the same seeded inputs, at sizes the oracle finishes in seconds that
still span several 64-token tiles, several split-KV chunks and ragged tails."""
import numpy as np
import pytest

import synth
from _harness import (assert_state_equal, check_attn, make_oracle, make_spork, pool_dims)

pytestmark = pytest.mark.gpu


def _build_both(cfg, k_per_seq=None, extra_pages=64, interleave=True):
    wl = synth.Workload(cfg, k_per_seq)
    npg, ms, mp = pool_dims(wl, extra_pages)
    orc = make_oracle(cfg, npg, ms, mp)
    spk = make_spork(cfg, npg, ms, mp)
    ids_o = synth.build_state(orc, wl, interleave)
    ids_s = synth.build_state(spk, wl, interleave)
    assert np.array_equal(ids_o, ids_s)
    return wl, orc, spk, ids_o


# ---------------------------------------------------------------------------
# config 1 (BASELINE.json configs[0]): tiny fork group, fp32, both phases of A-20
# ---------------------------------------------------------------------------
def test_cfg1_state_decode_and_fork_tail():
    cfg = synth.CFG1
    wl, orc, spk, ids = _build_both(cfg)
    assert_state_equal(orc, spk, ids)
    q = wl.q_all()
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "f32", "cfg1 decode")
    info = spk.last_plan()
    assert info["kernel"] == 0 and info["n_prefix_items"] >= 1
    assert info["unique_tokens"] == wl.unique_tokens() and info["naive_tokens"] == wl.naive_tokens()

    # phase B (A-20): fork the main stream at an unaligned length -> tail page duplicated
    main = int(ids[0])
    L = int(wl.total_len[0])
    if L % 16 == 0:
        r = synth.rng(1, synth.T_MISC, 0)
        k5 = synth.to_storage(r.standard_normal((5, cfg.Hkv, cfg.D), dtype=np.float32), "f32")
        v5 = synth.to_storage(r.standard_normal((5, cfg.Hkv, cfg.D), dtype=np.float32), "f32")
        orc.append([main], [5], k5, v5)
        spk.append([main], [5], k5, v5)
        L += 5
    ch_o = orc.fork([main])
    ch_s = spk.fork([main])
    assert np.array_equal(ch_o, ch_s)
    child = int(ch_s[0])
    assert_state_equal(orc, spk, list(ids) + [child])
    Lc, Tc = spk.export(child)
    Lm, Tm = spk.export(main)
    assert Lc == Lm == L and np.array_equal(Tc[:L // 16], Tm[:L // 16]) and Tc[L // 16] != Tm[L // 16]
    # tail valid slots bit-equal (and equal to the oracle's)
    t0 = (L // 16) * 16
    kc, vc = spk.read_kv(child, t0, L - t0)
    km, vm = spk.read_kv(main, t0, L - t0)
    ko, vo = orc.read_kv(child, t0, L - t0)
    assert np.array_equal(kc, km) and np.array_equal(vc, vm)
    assert np.array_equal(kc, ko) and np.array_equal(vc, vo)
    # a fork with an empty suffix decodes exactly like its parent
    q2 = np.concatenate([q[0:1], q[0:1]], axis=0)
    out2, lse2 = spk.decode_attn([0, 2], [main, child], q2)
    o2, l2 = out2.cpu().numpy(), lse2.cpu().numpy()
    ref2, lref2 = orc.decode([main, child], q2)
    check_attn(out2, lse2, ref2, lref2, "f32", "cfg1 fork pair")
    assert np.array_equal(o2[0], o2[1]) and np.array_equal(l2[0], l2[1])
    # release everything: refcounts return to zero
    everyone = list(ids) + [child]
    orc.release(everyone)
    spk.release(everyone)
    rc = spk.export_refcounts()
    assert np.array_equal(rc, orc.export_refcounts()) and not rc.any()
    assert spk.free_pages() == spk.num_pages and spk.status() == 0


# ---------------------------------------------------------------------------
# scaled-down bf16 decode configs (MMA path): several tiles, chunks, ragged tails
# ---------------------------------------------------------------------------
SMALL_DECODE = [
    # shapes of cfg 2 / 3 / 5 with short prefixes; prefix 1000 is not page aligned (tail copy at fork)
    synth.CFG2.scaled(n_groups=3, prefix_len=1000, suffix_lo=1, suffix_hi=300),
    synth.CFG3.scaled(n_groups=2, prefix_len=1536, suffix_lo=1, suffix_hi=260),
    synth.CFG5.scaled(n_groups=2, prefix_len=2048 + 16, suffix_lo=1, suffix_hi=200),
    # group of 3 (24 rows -> two row tiles, one half empty), tiny prefix
    synth.CFG3.scaled(n_groups=2, group_size=3, prefix_len=48, suffix_lo=0, suffix_hi=40),
    # group of 5 with G = 16: 80 rows -> two row blocks
    synth.CFG2.scaled(Hq=64, Hkv=4, n_groups=1, group_size=5, prefix_len=640, suffix_lo=0, suffix_hi=90),
]


# planner knob: which segments run on the tcgen05 kernel (None = default threshold)
PATHS = {"auto": None, "tcgen05": 1, "tcgen05-two-pipe": 1, "tcgen05-split-row": 1, "mma.sync": 1 << 20}


def _set_path(spk, path):
    if PATHS[path] is not None:
        spk.set_tensor_path_min_rows(PATHS[path])
    if path == "tcgen05-two-pipe":
        spk.set_many_row_variant(1)
    if path == "tcgen05-split-row":
        spk.set_many_row_variant(2)


def _check_kernel(info, path):
    if path.startswith("tcgen05"):
        assert info["kernel"] == 2 and info["n_umma_items"] == info["n_items"]
        if path == "tcgen05":
            assert info["n_two_pipe_items"] == 0
    elif path == "mma.sync":
        assert info["kernel"] == 1 and info["n_umma_items"] == 0
    else:
        assert info["kernel"] in (1, 2, 3)


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("cfg", SMALL_DECODE, ids=lambda c: f"{c.name}-g{c.group_size}-P{c.prefix_len}")
def test_small_bf16_decode(cfg, path):
    wl, orc, spk, ids = _build_both(cfg)
    _set_path(spk, path)
    assert_state_equal(orc, spk, ids)
    q = wl.q_all()
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "bf16", cfg.name)
    info = spk.last_plan()
    _check_kernel(info, path)
    if path in ("auto", "tcgen05"):
        # every segment is one row block -> stream-K schedule; the chunked LPT schedule gives the same
        # result up to the rounding of a different split
        assert info["stream_k"] == 1
        spk.set_stream_k(False)
        out_c, lse_c = spk.decode_attn(wl.group_indptr(), ids, q)
        assert spk.last_plan()["stream_k"] == 0
        check_attn(out_c, lse_c, out_ref, lse_ref, "bf16", cfg.name + " chunked schedule")
        spk.set_stream_k(True)
    # an unaligned fork point duplicates the tail page: those tokens are private copies
    dup = cfg.n_groups * (cfg.group_size - 1) * (cfg.prefix_len % 16)
    assert info["unique_tokens"] == wl.unique_tokens() + dup
    # invariant 1 on the GPU: the grouping only changes rounding
    out1, lse1 = spk.decode_attn(np.arange(len(ids) + 1), ids, q)
    check_attn(out1, lse1, out_ref, lse_ref, "bf16", cfg.name + " ungrouped")
    assert spk.last_plan()["n_prefix_items"] == 0
    # second call with nothing changed reuses the plan and gives identical bits
    out_b, lse_b = spk.decode_attn(np.arange(len(ids) + 1), ids, q)
    assert spk.last_plan()["plan_cached"] == 1
    assert np.array_equal(out1.cpu().numpy(), out_b.cpu().numpy())


@pytest.mark.parametrize("path", ["tcgen05", "tcgen05-two-pipe", "tcgen05-split-row", "mma.sync"])
@pytest.mark.parametrize("frac,scale", [(0.01, 8.0), (0.05, 16.0), (0.3, 4.0)])
def test_outlier_keys_running_max_jumps(frac, scale, path):
    """Attention-sink outliers (BASELINE.json config 3): the running row max jumps by far more than
    the tcgen05 kernel's lazy-rescale threshold in the middle of an item, so O is rescaled in TMEM;
    near-one-hot rows must still come out within tolerance."""
    cfg = synth.CFG3.scaled(n_groups=2, prefix_len=1040, suffix_lo=1, suffix_hi=150,
                            outlier_frac=frac, outlier_scale=scale)
    wl, orc, spk, ids = _build_both(cfg)
    _set_path(spk, path)
    q = wl.q_all()
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "bf16", f"outliers {frac} x{scale}")
    # the same through verify (k = 6 drafts per sequence, causal tail; 4 x 6 x 8 = 192 prefix rows:
    # two-pipe items on the tcgen05 path)
    kk = np.full(cfg.n_seqs, 6)
    cfgv = cfg.scaled(k_draft=6)
    wl, orc, spk, ids = _build_both(cfgv, kk)
    _set_path(spk, path)
    q, qi = wl.q_all(), wl.q_indptr()
    out_ref, lse_ref = orc.verify(ids, qi, q)
    out, lse = spk.verify_attn(wl.group_indptr(), ids, qi, q)
    check_attn(out, lse, out_ref, lse_ref, "bf16", f"verify outliers {frac} x{scale}")


def test_small_fp32_generic_paths():
    # fp32 D = 128 and bf16 D = 64 go through the simt kernel
    for cfg in (synth.CFG1.scaled(D=128, Hq=8, Hkv=2, prefix_len=200, suffix_hi=70),
                synth.CFG2.scaled(D=64, n_groups=2, prefix_len=330, suffix_lo=0, suffix_hi=100)):
        wl, orc, spk, ids = _build_both(cfg)
        assert_state_equal(orc, spk, ids)
        q = wl.q_all()
        out_ref, lse_ref = orc.decode(ids, q)
        out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
        check_attn(out, lse, out_ref, lse_ref, cfg.dtype, cfg.name)
        assert spk.last_plan()["kernel"] == 0


# ---------------------------------------------------------------------------
# verify (config 4 shape, scaled): mixed k, causal within the drafts
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("ks", [[4, 8, 16, 1], [16, 16, 16, 16], [1, 1, 1, 1], [3, 7, 12, 5]])
def test_small_verify(ks, path):
    cfg = synth.CFG4.scaled(n_groups=2, prefix_len=1024 + 32, suffix_lo=0, suffix_hi=100)
    kk = np.array(ks * cfg.n_groups)
    wl, orc, spk, ids = _build_both(cfg, kk)
    _set_path(spk, path)
    assert_state_equal(orc, spk, ids)
    q, qi = wl.q_all(), wl.q_indptr()
    out_ref, lse_ref = orc.verify(ids, qi, q)
    out, lse = spk.verify_attn(wl.group_indptr(), ids, qi, q)
    check_attn(out, lse, out_ref, lse_ref, "bf16", f"verify k={ks}")
    _check_kernel(spk.last_plan(), path)
    if path in ("tcgen05-two-pipe", "tcgen05-split-row"):
        # a group of 4 with G = 8: the shared prefix has 32 * mean(k) rows -> two-pipe items iff > 128
        assert (spk.last_plan()["n_two_pipe_items"] > 0) == (32 * sum(ks) // 4 > 128)
    # ungrouped = same result
    out1, lse1 = spk.verify_attn(np.arange(len(ids) + 1), ids, qi, q)
    check_attn(out1, lse1, out_ref, lse_ref, "bf16", f"verify ungrouped k={ks}")
    # k = 1 everywhere is decode
    if set(ks) == {1}:
        out_d, lse_d = spk.decode_attn(wl.group_indptr(), ids, q)
        assert np.array_equal(out_d.cpu().numpy(), out.cpu().numpy())


def test_verify_fp32_and_errors():
    cfg = synth.CFG1.scaled(k_draft=5, prefix_len=100, suffix_hi=20)
    wl, orc, spk, ids = _build_both(cfg)
    q, qi = wl.q_all(), wl.q_indptr()
    out_ref, lse_ref = orc.verify(ids, qi, q)
    out, lse = spk.verify_attn(wl.group_indptr(), ids, qi, q)
    check_attn(out, lse, out_ref, lse_ref, "f32", "verify fp32")
    import paper_2607_03333_b200 as sp
    # k > len and k < 1 are rejected; so are dead sequences
    bad = qi.copy()
    bad[1:] += 1000
    rc, _, _ = spk.verify_attn(wl.group_indptr(), ids, bad, np.zeros((int(bad[-1]), cfg.Hq, cfg.D), np.float32),
                               check=False)
    assert rc == sp.ERR_INVALID
    rc, _, _ = spk.verify_attn(wl.group_indptr(), ids, np.zeros_like(qi), q, check=False)
    assert rc == sp.ERR_INVALID
    rc, _, _ = spk.decode_attn([0, 1], [7], q[:1], check=False)
    assert rc == sp.ERR_INVALID_SEQ


# ---------------------------------------------------------------------------
# degenerate cases
# ---------------------------------------------------------------------------
def test_degenerate_groups():
    cfg = synth.CFG2.scaled(n_groups=2, prefix_len=256, suffix_lo=0, suffix_hi=0)  # empty suffixes
    wl, orc, spk, ids = _build_both(cfg)
    q = wl.q_all()
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "bf16", "empty suffix")
    # members of one group that share nothing (declared group of unrelated sequences)
    mixed = np.array([ids[0], ids[2]], np.int32)
    qm = np.stack([q[0], q[2]])
    o_ref, l_ref = orc.decode(mixed, qm)
    o, l = spk.decode_attn([0, 2], mixed, qm)
    check_attn(o, l, o_ref, l_ref, "bf16", "unrelated members")
    assert spk.last_plan()["n_prefix_items"] == 0
    # an empty sequence: out = 0, lse = -inf; one token: out = V (single key returns its V)
    e_o, e_s = orc.seq_create(2), spk.seq_create(2)
    assert np.array_equal(e_o, e_s)
    r = synth.rng(2, synth.T_MISC, 1)
    k1 = synth.to_storage(r.standard_normal((1, cfg.Hkv, cfg.D), dtype=np.float32), "bf16")
    v1 = synth.to_storage(r.standard_normal((1, cfg.Hkv, cfg.D), dtype=np.float32), "bf16")
    orc.append(e_o[1:], [1], k1, v1)
    spk.append(e_s[1:], [1], k1, v1)
    qe = q[:2]
    o, l = spk.decode_attn([0, 1, 2], e_s, qe)
    o, l = o.cpu().numpy(), l.cpu().numpy()
    assert not o[0].any() and np.all(np.isneginf(l[0]))
    vf = synth.bf16_bits_to_f32(v1)[0]          # [Hkv][D]
    for h in range(cfg.Hq):
        assert np.array_equal(o[1, h], vf[h // cfg.G])
    o_ref, l_ref = orc.decode(e_o, qe)
    assert np.allclose(l[1], l_ref[1], rtol=1e-4, atol=1e-4)


def test_parent_released_before_children():
    cfg = synth.CFG3.scaled(n_groups=1, prefix_len=512, suffix_lo=5, suffix_hi=60)
    wl, orc, spk, ids = _build_both(cfg)
    q = wl.q_all()
    orc.release(ids[:1])
    spk.release(ids[:1])
    assert_state_equal(orc, spk, ids[1:])
    out_ref, lse_ref = orc.decode(ids[1:], q[1:])
    out, lse = spk.decode_attn([0, len(ids) - 1], ids[1:], q[1:])
    check_attn(out, lse, out_ref, lse_ref, "bf16", "children after parent release")
    assert spk.last_plan()["n_prefix_items"] >= 1
    orc.release(ids[1:])
    spk.release(ids[1:])
    assert not spk.export_refcounts().any()


# ---------------------------------------------------------------------------
# fragmented pool (dummy sequences pin a random half of the pool)
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("path", ["auto", "mma.sync"])
def test_fragmented_pool(path):
    """Dummy sequences fill the pool, a random half of them is released, and the workload is built into
    the holes: block tables are scattered page ids (lowest free id first, A-1), bit-exact on both
    sides, and attention over them matches the oracle."""
    cfg = synth.CFG5.scaled(n_groups=2, group_size=3, prefix_len=900, suffix_lo=1, suffix_hi=260)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 64)
    n_dummy = 120
    orc = make_oracle(cfg, npg + n_dummy * 3, ms + n_dummy, mp)
    spk = make_spork(cfg, npg + n_dummy * 3, ms + n_dummy, mp)
    _set_path(spk, path)
    r = np.random.default_rng(31)
    dummies = orc.seq_create(n_dummy)
    assert np.array_equal(dummies, spk.seq_create(n_dummy))
    for s in dummies:                       # 1..3 pages each, interleaved
        n = int(r.integers(1, 3 * 16 + 1))
        k = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
        orc.append([s], [n], k, k)
        spk.append([s], [n], k, k)
    gone = r.permutation(dummies)[: n_dummy // 2]
    orc.release(gone)
    spk.release(gone)
    ids = synth.build_state(orc, wl)
    assert np.array_equal(ids, synth.build_state(spk, wl))
    assert_state_equal(orc, spk, ids)
    L, T = spk.export(int(ids[0]))
    assert np.any(np.diff(T) != 1)          # really scattered
    q = wl.q_all()
    out_ref, lse_ref = orc.decode(ids, q)
    out, lse = spk.decode_attn(wl.group_indptr(), ids, q)
    check_attn(out, lse, out_ref, lse_ref, "bf16", "fragmented pool")
    assert spk.last_plan()["n_prefix_items"] >= 1
