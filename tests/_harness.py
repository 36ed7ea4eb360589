"""Shared helpers of the GPU parity tests: build the same seeded state in the CPU
oracle and in libspork (through the C ABI), and compare.

Tolerances (BASELINE.json `north_star`):
  block tables, lengths, refcounts: bit-exact
  out:  max abs error <= 1e-5 (fp32 KV), <= 1e-2 (bf16 KV, fp32 accumulation)
  lse:  |d| <= 1e-4 * max(1, |lse*|)   (reading A-21)
"""
from __future__ import annotations

import numpy as np

import oracle
import synth

OUT_TOL = {"f32": 1e-5, "bf16": 1e-2, "e4m3": 1e-2}    # e4m3 KV: DESIGN.md section 6
LSE_RTOL = 1e-4


def make_oracle(cfg: synth.SporkConfig, num_pages: int, max_seqs: int, max_pages: int, store_kv=True):
    return oracle.Oracle(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, num_pages, max_seqs, max_pages, cfg.scale,
                         store_kv=store_kv)


def make_spork(cfg: synth.SporkConfig, num_pages: int, max_seqs: int, max_pages: int):
    import paper_2607_03333_b200 as sp
    return sp.Spork(cfg.dtype, cfg.Hq, cfg.Hkv, cfg.D, num_pages, max_seqs, max_pages, cfg.scale)


def pool_dims(wl: synth.Workload, slack_pages: int = 64):
    c = wl.cfg
    per_seq = int((wl.total_len.max() + c.page_size - 1) // c.page_size) + 2
    total = int(c.n_groups * ((c.prefix_len + 15) // 16) +
                sum((int(x) + 15) // 16 + 1 for x in wl.private_len)) + c.n_seqs + slack_pages
    return total, c.n_seqs + 8, per_seq


class Both:
    """synth.build_state engine that replays every call on the oracle AND on libspork (the generated
    K/V values are produced once), checking that both hand out the same ids."""

    def __init__(self, orc, spk):
        self.orc, self.spk = orc, spk

    def seq_create(self, n):
        a, b = self.orc.seq_create(n), self.spk.seq_create(n)
        assert np.array_equal(a, b)
        return a

    def append(self, seq_ids, n_tokens, k, v):
        self.orc.append(seq_ids, n_tokens, k, v)
        self.spk.append(seq_ids, n_tokens, k, v)

    def fork(self, parents):
        a, b = self.orc.fork(parents), self.spk.fork(parents)
        assert np.array_equal(a, b)
        return a

    def release(self, seq_ids):
        self.orc.release(seq_ids)
        self.spk.release(seq_ids)

    def truncate(self, seq_ids, new_len):
        self.orc.truncate(seq_ids, new_len)
        self.spk.truncate(seq_ids, new_len)


def assert_state_equal(orc, spk, seq_ids, check_kv_tail=True):
    """bit-exact lengths, block tables and refcounts (device vs oracle)."""
    for s in seq_ids:
        Lo, To = orc.export_seq(int(s))
        Ls, Ts = spk.export(int(s))
        assert Lo == Ls, f"len of seq {s}: oracle {Lo} device {Ls}"
        assert np.array_equal(To, Ts), f"block table of seq {s} differs"
    assert np.array_equal(orc.export_refcounts(), spk.export_refcounts()), "refcounts differ"
    assert spk.status() == 0


def check_attn(out_dev, lse_dev, out_ref, lse_ref, dtype: str, what: str = ""):
    out = out_dev.detach().cpu().numpy().astype(np.float64)
    lse = lse_dev.detach().cpu().numpy().astype(np.float64)
    assert out.shape == out_ref.shape and lse.shape == lse_ref.shape
    assert np.all(np.isfinite(out)), f"{what}: non-finite out"
    err = float(np.max(np.abs(out - out_ref))) if out.size else 0.0
    assert err <= OUT_TOL[dtype], f"{what}: max abs err {err:.3e} > {OUT_TOL[dtype]}"
    fin = np.isfinite(lse_ref)
    assert np.array_equal(fin, np.isfinite(lse)), f"{what}: lse finiteness differs"
    if fin.any():
        rel = np.abs(lse[fin] - lse_ref[fin]) / np.maximum(1.0, np.abs(lse_ref[fin]))
        assert float(rel.max()) <= LSE_RTOL, f"{what}: lse rel err {float(rel.max()):.3e}"
    return err


def sampled_rows_check(spk_out, spk_lse, wl: synth.Workload, samples, what=""):
    """Full-size configs: compare sampled (seq, q row j, head) outputs with the
    oracle's dense plain-definition routine on regenerated K/V."""
    c = wl.cfg
    qi = wl.q_indptr()
    out = spk_out.detach().cpu().numpy().astype(np.float64)
    lse = spk_lse.detach().cpu().numpy().astype(np.float64)
    worst = 0.0
    cache = {}
    for (seq, j, h) in samples:
        if seq not in cache:
            cache.clear()
            cache[seq] = (wl.dense_kv(seq), wl.q(seq))
        (K, V), Q = cache[seq]
        L, k = int(wl.total_len[seq]), int(wl.k[seq])
        n_att = L if k == 0 else L - k + j + 1
        kvh = h // c.G
        o_ref, l_ref = oracle.attend_dense(c.dtype, c.scale, Q[j, h], K[:n_att, kvh], V[:n_att, kvh])
        row = int(qi[seq]) + j
        err = float(np.max(np.abs(out[row, h] - o_ref)))
        worst = max(worst, err)
        assert err <= OUT_TOL[c.dtype], f"{what} seq {seq} row {j} head {h}: err {err:.3e}"
        assert abs(lse[row, h] - l_ref) <= LSE_RTOL * max(1.0, abs(l_ref)), \
            f"{what} seq {seq} row {j} head {h}: lse {lse[row, h]} vs {l_ref}"
    return worst
