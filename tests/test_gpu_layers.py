"""Multi-layer step, SURVEY 8(f) NEXT-4 (the Qwen3 models of PAPER.md:299 have 36 / 64 / 48 layers):
one handle, one set of block tables / refcounts, L pairs of K/V pools, ONE plan and L back-to-back
(attention, merge) launches.  The oracle is one plain single-layer instance per layer, driven by the
same call script -- layers are independent in the definition."""
import numpy as np
import pytest

import synth
from _harness import assert_state_equal, check_attn, make_oracle, make_spork, pool_dims

pytestmark = pytest.mark.gpu


class Layered:
    """engine for synth.build_state: layer 0 gets the generated values, layer l a deterministic
    transform of them (sign flips / a roll along D), on both sides."""

    def __init__(self, orcs, spk):
        self.orcs, self.spk, self.L = orcs, spk, len(orcs)

    @staticmethod
    def variant(x, l):
        if l == 0:
            return x
        y = np.roll(x, l, axis=-1).copy()
        if l % 2:
            y ^= np.uint16(0x8000)          # flip the bf16 sign bit
        return y

    def seq_create(self, n):
        ids = [o.seq_create(n) for o in self.orcs]
        s = self.spk.seq_create(n)
        assert all(np.array_equal(i, s) for i in ids)
        return s

    def append(self, seq_ids, n_tokens, k, v):
        for l, o in enumerate(self.orcs):
            o.append(seq_ids, n_tokens, self.variant(k, l), self.variant(v, l))
        self.spk.append(seq_ids, n_tokens, k, v)
        for l in range(1, self.L):
            self.spk.write_kv_layer(l, seq_ids, n_tokens, self.variant(k, l), self.variant(v, l))

    def fork(self, parents):
        ch = [o.fork(parents) for o in self.orcs]
        s = self.spk.fork(parents)
        assert all(np.array_equal(c, s) for c in ch)
        return s


@pytest.mark.parametrize("verify", [False, True])
def test_layers_parity(verify):
    import torch
    L = 5
    cfg = synth.CFG2.scaled(n_groups=3, prefix_len=1000, suffix_lo=1, suffix_hi=200, k_draft=6 if verify else 0)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 64)
    orcs = [make_oracle(cfg, npg, ms, mp) for _ in range(L)]
    spk = make_spork(cfg, npg, ms, mp)
    spk.layers(L)
    ids = synth.build_state(Layered(orcs, spk), wl)          # prefix 1000: forks duplicate a tail page in every layer
    assert_state_equal(orcs[0], spk, ids)
    gi, qi = wl.group_indptr(), wl.q_indptr()
    q0 = wl.q_all()
    qs = [spk._dev(Layered.variant(q0, l)) for l in range(L)]
    rows = q0.shape[0]
    outs = [torch.empty((rows, cfg.Hq, cfg.D), dtype=torch.float32, device=spk.device) for _ in range(L)]
    lses = [torch.empty((rows, cfg.Hq), dtype=torch.float32, device=spk.device) for _ in range(L)]
    for rep in range(2):                                     # the second call reuses the plan
        for o in outs:
            o.fill_(float("nan"))
        spk.attn_layers(gi, ids, qs, outs, lses, qi if verify else None)
        info = spk.last_plan()
        assert info["launches"] == 2 * L and info["plan_cached"] == rep
        for l in range(L):
            ql = Layered.variant(q0, l)
            ref, lref = orcs[l].verify(ids, qi, ql) if verify else orcs[l].decode(ids, ql)
            check_attn(outs[l], lses[l], ref, lref, "bf16", f"layer {l}")
    # single-layer calls on layer 0 still work and agree bit for bit with the multi-layer result
    o1, l1 = (spk.verify_attn(gi, ids, qi, qs[0]) if verify else spk.decode_attn(gi, ids, qs[0]))
    assert np.array_equal(o1.cpu().numpy(), outs[0].cpu().numpy())
    # tail pages were duplicated in every layer: a fork child reads its own copy
    k_l, v_l = spk.read_kv(int(ids[1]), 992, 8)
    ko, vo = orcs[0].read_kv(int(ids[1]), 992, 8)
    assert np.array_equal(k_l, ko) and np.array_equal(v_l, vo)


def test_layers_argument_errors():
    import paper_2607_03333_b200 as sp
    import ctypes as C
    cfg = synth.CFG2.scaled(n_groups=1, prefix_len=64, suffix_lo=1, suffix_hi=5)
    wl = synth.Workload(cfg)
    npg, ms, mp = pool_dims(wl, 16)
    spk = make_spork(cfg, npg, ms, mp)
    ids = synth.build_state(spk, wl)
    # no layers registered: a 2-layer call is rejected, write_kv_layer(1) too
    two = (C.c_void_p * 2)(0, 0)
    gi = np.array([0, 2], np.int32)
    rc = spk.lib.spork_decode_attn_layers(spk._h, 2, 1, gi.ctypes.data_as(C.c_void_p), ids.ctypes.data_as(C.c_void_p),
                                          two, two, two, spk._st)
    assert rc == sp.ERR_INVALID
    k = np.zeros((2, cfg.Hkv, cfg.D), np.uint16)
    assert spk.write_kv_layer(1, ids, [1, 1], k, k, check=False) == sp.ERR_INVALID
    spk.layers(2)
    assert spk.write_kv_layer(1, ids, [1, 10**6], k, k, check=False) == sp.ERR_INVALID
    assert spk.write_kv_layer(1, ids, [1, 1], k, k, check=False) == 0
