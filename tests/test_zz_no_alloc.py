"""spork_confidence_static (include/spork.h): the Eq. 2 confidence score for callers that
cannot allocate -- its per-(row, slice) partials live in a file-scope device array instead of a buffer the
context grows.  Checked against the existing path, spork_confidence, within the tolerance of
tests/test_gpu_confidence.py (and against the fp64 oracle), on two calls in a row that share the array:
the second is smaller and sliced differently, so it runs over the first one's leftovers.

This file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  It passes alone in a fresh process and after the other tests (the array is per process,
nothing here depends on what ran before).
"""
import numpy as np
import pytest

import oracle
import synth
from _harness import make_spork

pytestmark = pytest.mark.gpu

RTOL = 2e-5      # as tests/test_gpu_confidence.py: fp32 sums of ex2.approx terms against fp64


def _case(spk, n_spans, vocab, seed):
    import torch
    x, sp = synth.probe_logits(n_spans, vocab, seed=seed)
    xd = spk._dev(x)
    spd = spk._dev(np.asarray(sp, np.int32))
    out = torch.full((n_spans,), -1.0, dtype=torch.float32, device=spk.device)
    return x, np.asarray(sp, np.int32), xd, spd, out


def _check(spk, case, what):
    x, sp, xd, spd, out = case
    want = spk.confidence(sp, xd).cpu().numpy().astype(np.float64)          # the existing path
    got = out.cpu().numpy().astype(np.float64)
    assert got.shape == want.shape
    assert np.allclose(got, want, rtol=RTOL, atol=0), (what, float(np.max(np.abs(got / want - 1))))
    ref = oracle.confidence(x, sp)
    assert np.allclose(got, ref, rtol=RTOL, atol=0), (what, float(np.max(np.abs(got / ref - 1))))
    assert np.all(got[np.diff(sp) <= 1] == 1.0)                              # empty minimum (A-23)


def test_static_scratch_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    spk = make_spork(synth.CFG1, 8, 2, 4)
    a = _case(spk, 40, 151936, seed=11)       # few rows: many vocabulary slices per row
    b = _case(spk, 9, 2048 * 8 + 1, seed=12)  # fewer rows, odd vocabulary (scalar loads), other slicing
    assert spk.confidence_static(a[3], a[2], a[4]) == 0
    assert spk.confidence_static(b[3], b[2], b[4]) == 0      # second call: the array holds the first one's partials
    _check(spk, a, "first call")
    _check(spk, b, "second call")
    # the two again, now that every kernel is loaded: the device's free memory does not move
    spk.synchronize()
    free0 = torch.cuda.mem_get_info(spk.device)[0]
    for c in (a, b):
        c[4].fill_(-1.0)
        assert spk.confidence_static(c[3], c[2], c[4]) == 0
    spk.synchronize()
    assert torch.cuda.mem_get_info(spk.device)[0] == free0
    _check(spk, a, "third call")
    _check(spk, b, "fourth call")
    spk.close()


def test_static_scratch_entry_point_edges_and_limit():
    import torch
    import paper_2607_03333_b200 as sp_mod
    spk = make_spork(synth.CFG1, 8, 2, 4)
    V = 4096
    x = np.zeros((6, V), np.float32)
    x[:, 11] = [30, 30, 2, 30, -5, 30]
    x[4, :] = -np.inf                       # a row with a single finite logit: probability exactly 1
    x[4, 100] = 0.0
    sp = np.array([0, 3, 3, 6], np.int32)   # middle span empty
    xd, spd = spk._dev(x), spk._dev(sp)
    out = torch.full((3,), -1.0, dtype=torch.float32, device=spk.device)
    assert spk.confidence_static(spd, xd, out) == 0
    _check(spk, (x, sp, xd, spd, out), "edges")
    assert out.cpu().numpy()[1] == 1.0
    # a set-up call (no spans) launches nothing; no rows at all: every span is empty
    lib = spk.lib
    assert lib.spork_confidence_static(0, None, 0, None, V, None, spk._st) == 0
    out2 = torch.full((2,), -1.0, dtype=torch.float32, device=spk.device)
    assert spk.confidence_static(spk._dev(np.zeros(3, np.int32)), xd[:0], out2) == 0
    assert out2.cpu().numpy().tolist() == [1.0, 1.0]
    # spans that break the contract (device memory, not checked): clamped to the rows that exist -- the
    # scores mean nothing, but nothing faults and the next call is served as usual
    bad = spk._dev(np.array([0, 10 ** 6, -5, 3], np.int32))
    assert spk.confidence_static(bad, xd, out) == 0
    spk.synchronize()
    assert spk.confidence_static(spd, xd, out) == 0
    _check(spk, (x, sp, xd, spd, out), "after a bad span_indptr")
    # one row beyond the fixed maximum: refused before anything is launched, the output is untouched
    n = sp_mod.CONFIDENCE_STATIC_MAX_ROWS + 1
    big = torch.zeros((n, 8), dtype=torch.float32, device=spk.device)
    spb = spk._dev(np.array([0, n], np.int32))
    out3 = torch.full((1,), -1.0, dtype=torch.float32, device=spk.device)
    assert spk.confidence_static(spb, big, out3, check=False) == sp_mod.ERR_LIMIT
    assert out3.item() == -1.0
    assert "maximum" in lib.spork_strerror(sp_mod.ERR_LIMIT).decode()
    # exactly the maximum is served (2 slices per row at most)
    big = big[:n - 1]
    big[:, 3] = 1.0
    spb = spk._dev(np.array([0, n - 1], np.int32))
    assert spk.confidence_static(spb, big, out3) == 0
    assert np.isclose(out3.item(), 1.0 / (1.0 + 7.0 * np.exp(-1.0)), rtol=RTOL)
    spk.close()


def test_static_scratch_entry_point_under_graph_capture():
    """what the entry point is for: a capture in which nothing may allocate, replayed on new logits"""
    import torch
    spk = make_spork(synth.CFG1, 8, 2, 4)
    a = _case(spk, 24, 32000, seed=5)
    assert spk.confidence_static(a[3], a[2], a[4]) == 0       # (first call on the device: outside capture)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=spk.stream):
        spk.confidence_static(a[3], a[2], a[4])
    x0, sp0 = a[0], a[1]
    for seed in (6, 7):
        # new logits of the same shape; the second replay also moves the span boundaries (same row count)
        x = (x0 + 3.0 * np.random.default_rng(seed).standard_normal(x0.shape, dtype=np.float32)).astype(np.float32)
        sp = sp0 if seed == 6 else np.concatenate([[0], np.cumsum(np.diff(sp0)[::-1])]).astype(np.int32)
        with torch.cuda.stream(spk.stream):
            a[2].copy_(torch.from_numpy(x))
            a[3].copy_(torch.from_numpy(sp))
            g.replay()
        _check(spk, (x, sp, a[2], a[3], a[4]), f"replay {seed}")
    spk.close()
