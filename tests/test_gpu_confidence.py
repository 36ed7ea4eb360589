"""GPU parity of spork_confidence (Eq. 2) against the fp64 oracle."""
import numpy as np
import pytest

import oracle
import synth
from _harness import make_spork

pytestmark = pytest.mark.gpu

RTOL = 2e-5      # fp32 sums of ex2.approx terms (2^-22 each) against fp64


@pytest.mark.parametrize("vocab,n_spans", [(151936, 24), (32000, 7), (1003, 40), (5, 3), (2048 * 8 + 1, 9)])
def test_confidence_matches_oracle(vocab, n_spans):
    spk = make_spork(synth.CFG1, 8, 2, 4)
    x, sp = synth.probe_logits(n_spans, vocab, seed=vocab % 97)
    want = oracle.confidence(x, sp)
    got = spk.confidence(sp, x).cpu().numpy().astype(np.float64)
    assert got.shape == want.shape
    assert np.allclose(got, want, rtol=RTOL, atol=0), float(np.max(np.abs(got / want - 1)))
    assert np.all(got[np.diff(sp) <= 1] == 1.0)                       # empty minimum (A-23)
    assert 0 < got.min() and got.max() <= 1.0


def test_confidence_edges():
    import paper_2607_03333_b200 as sp_mod
    spk = make_spork(synth.CFG1, 8, 2, 4)
    V = 4096
    x = np.zeros((6, V), np.float32)
    x[:, 11] = [30, 30, 2, 30, -5, 30]
    x[4, :] = -np.inf                      # a row with a single finite logit: probability exactly 1
    x[4, 100] = 0.0
    sp = np.array([0, 3, 3, 6], np.int32)   # middle span empty
    got = spk.confidence(sp, x).cpu().numpy()
    want = oracle.confidence(x, sp)
    assert np.allclose(got, want, rtol=RTOL) and got[1] == 1.0          # empty span: exactly 1
    assert spk.confidence(np.array([0], np.int32), np.zeros((0, V), np.float32)).numel() == 0
    rc, _ = spk.confidence(np.array([0, 2, 1], np.int32), x, check=False)
    assert rc == sp_mod.ERR_INVALID
