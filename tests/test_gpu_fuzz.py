"""Randomised batch shapes against the oracle: groups of 1..5 members, prefixes of 0..700 tokens
(0: nothing shared), private tails of 0..180 tokens, forks of forks -- the shapes the planner's
stream-K partition and the chunked schedule have to cut, through every kernel path."""
import numpy as np
import pytest

import synth
from _harness import assert_state_equal, check_attn, make_oracle, make_spork

pytestmark = pytest.mark.gpu


def _kv(r, n, cfg):
    k = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
    v = synth.to_storage(r.standard_normal((n, cfg.Hkv, cfg.D), dtype=np.float32), cfg.dtype)
    return k, v


def _append(both, seq, n, r, cfg):
    if n > 0:
        k, v = _kv(r, n, cfg)
        for x in both:
            x.append([seq], [n], k, v)


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
@pytest.mark.parametrize("path", ["auto", "chunked", "mma.sync", "e4m3", "e4m3-chunked"])
def test_random_batches(seed, path):
    cfg = synth.CFG2.scaled(n_groups=1) if seed % 2 == 0 else synth.CFG5.scaled(n_groups=1)
    if path.startswith("e4m3"):
        cfg = cfg.scaled(dtype="e4m3")          # FP8-KV variant: e4m3 cache, bf16 queries
    r = np.random.default_rng([77, seed])
    orc, spk = make_oracle(cfg, 1024, 64, 80), make_spork(cfg, 1024, 64, 80)
    if path.endswith("chunked"):
        spk.set_stream_k(False)
    if path == "mma.sync":
        spk.set_tensor_path_min_rows(1 << 20)
    both = (orc, spk)
    indptr, seqs = [0], []
    for _ in range(int(r.integers(3, 9))):
        root = int(orc.seq_create(1)[0])
        assert int(spk.seq_create(1)[0]) == root
        _append(both, root, int(r.choice([0, 1, 15, 16, 17, int(r.integers(18, 700))])), r, cfg)
        members = [root]
        for _ in range(int(r.integers(0, 5))):
            parent = members[int(r.integers(0, len(members)))]      # forks of forks
            if orc.export_seq(parent)[0] == 0:
                continue
            co, cs = orc.fork([parent]), spk.fork([parent])
            assert np.array_equal(co, cs)
            members.append(int(cs[0]))
            _append(both, members[-1], int(r.integers(0, 60)), r, cfg)
        for m in members:
            _append(both, m, int(r.integers(0, 180)), r, cfg)
        seqs += members
        indptr.append(len(seqs))
    seqs = np.array(seqs, np.int32)
    assert_state_equal(orc, spk, seqs)
    q = synth.to_storage(r.standard_normal((len(seqs), cfg.Hq, cfg.D), dtype=np.float32), cfg.q_dtype)
    ref, lref = orc.decode(seqs, q)
    out, lse = spk.decode_attn(indptr, seqs, q)
    check_attn(out, lse, ref, lref, cfg.dtype, f"fuzz decode seed {seed}")
    info = spk.last_plan()
    assert info["stream_k"] == (1 if path in ("auto", "e4m3") else 0)
    # verify on the non-empty sequences with random draft counts (1 .. min(len, 9))
    lens = np.array([orc.export_seq(int(s))[0] for s in seqs])
    keep = lens > 0
    vs = seqs[keep]
    ks = np.minimum(r.integers(1, 10, size=len(vs)), lens[keep])
    qi = np.concatenate([[0], np.cumsum(ks)]).astype(np.int32)
    qv = synth.to_storage(r.standard_normal((int(qi[-1]), cfg.Hq, cfg.D), dtype=np.float32), cfg.q_dtype)
    ref, lref = orc.verify(vs, qi, qv)
    out, lse = spk.verify_attn(np.arange(len(vs) + 1), vs, qi, qv)      # every sequence its own group
    check_attn(out, lse, ref, lref, cfg.dtype, f"fuzz verify seed {seed}")
    for x in both:
        x.release(seqs)
    assert not spk.export_refcounts().any() and spk.status() == 0
