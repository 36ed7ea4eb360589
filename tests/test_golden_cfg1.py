"""tests/golden/cfg1_oracle.txt (config 1, BASELINE.json configs[0]) as a regression fixture.

The file was written by tests/golden/make_cfg1_golden.py from oracle/ and synth/ alone.  The CPU test
checks that today's oracle (and today's seeded inputs) still reproduce it -- a change to the oracle's
arithmetic, to the allocation policy (A-1) or to the input recipe shows up here; the GPU test holds the
CUDA path to the same stored values: block tables and refcounts bit-exact, out/lse within the fp32
tolerances of BASELINE.json `north_star`.
"""
import os

import numpy as np
import pytest

import oracle
import synth

PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg1_oracle.txt")


def load_fixture():
    fx = {"seq": {}, "lse": {}, "out": {}}
    with open(PATH) as f:
        for line in f:
            t = line.split()
            if not t or t[0].startswith("#"):
                continue
            if t[0] == "suffix_len":
                fx["suffix_len"] = [int(x) for x in t[1:]]
            elif t[0] == "seq":
                fx["seq"][int(t[1])] = (int(t[3]), np.array([int(x) for x in t[5:]], np.int32))
            elif t[0] == "refcount_nonzero":
                fx["refcount"] = {int(a): int(b) for a, b in (x.split(":") for x in t[1:])}
            elif t[0] == "lse":
                fx["lse"][(int(t[1]), int(t[2]))] = float(t[3])
            elif t[0] == "out":
                fx["out"][(int(t[1]), int(t[2]))] = np.array([float(x) for x in t[3:]])
    return fx


def check_state(fx, export_seq, refcounts):
    for s, (L, tab) in fx["seq"].items():
        Ls, Ts = export_seq(s)
        assert Ls == L and np.array_equal(np.asarray(Ts)[:len(tab)], tab), f"seq {s}"
    nz = {int(i): int(v) for i, v in enumerate(refcounts) if v}
    assert nz == fx["refcount"]


def test_oracle_reproduces_the_fixture():
    fx = load_fixture()
    c = synth.CFG1
    wl = synth.Workload(c)
    assert [int(x) for x in wl.suffix_len] == fx["suffix_len"]
    o = oracle.Oracle(c.dtype, c.Hq, c.Hkv, c.D, 64, 8, 32, c.scale)
    ids = synth.build_state(o, wl)
    assert sorted(int(s) for s in ids) == sorted(fx["seq"])
    check_state(fx, o.export_seq, o.export_refcounts())
    out, lse = o.decode(ids, wl.q_all())
    assert len(fx["lse"]) == out.shape[0] * out.shape[1]
    for (i, h), v in fx["lse"].items():
        assert abs(lse[i, h] - v) <= 1e-13 * max(1.0, abs(v))
        assert np.max(np.abs(out[i, h, :8] - fx["out"][(i, h)])) <= 1e-14


@pytest.mark.gpu
def test_cuda_path_matches_the_fixture():
    import paper_2607_03333_b200 as sp
    fx = load_fixture()
    c = synth.CFG1
    wl = synth.Workload(c)
    spk = sp.Spork(c.dtype, c.Hq, c.Hkv, c.D, 64, 8, 32, c.scale)
    ids = synth.build_state(spk, wl)
    check_state(fx, spk.export, spk.export_refcounts())
    out, lse = spk.decode_attn(wl.group_indptr(), ids, wl.q_all())
    out, lse = out.cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64)
    for (i, h), v in fx["lse"].items():
        assert abs(lse[i, h] - v) <= 1e-4 * max(1.0, abs(v))
        assert np.max(np.abs(out[i, h, :8] - fx["out"][(i, h)])) <= 1e-5
    spk.release(ids)
    assert not spk.export_refcounts().any()
    spk.close()
