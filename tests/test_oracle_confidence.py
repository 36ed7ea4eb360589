"""Pins of the oracle's D2 confidence score (Eq. 2: c = min_{i=2..L} exp(l_i), l_i the
top-1 log-probability) against closed forms and scipy's softmax."""
import numpy as np
from scipy.special import softmax

import oracle


def test_closed_forms():
    V = 1000
    # uniform logits: every token has probability 1/V -> c = 1/V, whatever the constant
    x = np.full((4, V), 3.25)
    assert np.allclose(oracle.confidence(x, [0, 4]), [1.0 / V], rtol=1e-12)
    # two tokens tied at the top with the rest far below: top-1 probability 1/2
    x = np.full((3, V), -1e3)
    x[:, 7] = x[:, 9] = 5.0
    assert np.allclose(oracle.confidence(x, [0, 3]), [0.5], rtol=1e-12)
    # one dominant token: p = 1 / (1 + (V-1) e^-d)
    d = 6.0
    x = np.zeros((2, V))
    x[:, 3] = d
    assert np.allclose(oracle.confidence(x, [0, 2]), [1.0 / (1.0 + (V - 1) * np.exp(-d))], rtol=1e-12)
    # the first row of a span is skipped; spans of one row (or none) give 1 (A-23)
    x = np.zeros((5, V))
    x[1:, 0] = 50.0                      # rows 1.. are confident, row 0 is uniform
    assert np.allclose(oracle.confidence(x, [0, 5]), [1.0], atol=1e-12)
    assert np.array_equal(oracle.confidence(x, [0, 1, 1, 2]), [1.0, 1.0, 1.0])
    # the minimum picks the least confident row of the span, and only of ITS span
    x = np.zeros((6, V))
    x[:, 0] = [9, 9, 2, 9, 9, 1]
    p = lambda dd: 1.0 / (1.0 + (V - 1) * np.exp(-dd))
    assert np.allclose(oracle.confidence(x, [0, 3, 6]), [p(2), p(1)], rtol=1e-12)


def test_matches_scipy_softmax_and_shift_invariance():
    r = np.random.default_rng(4)
    x = r.standard_normal((40, 777)) * 3
    sp = np.array([0, 4, 5, 12, 12, 30, 40])
    want = [softmax(x[a + 1:b], axis=1).max(axis=1).min() if b - a > 1 else 1.0 for a, b in zip(sp[:-1], sp[1:])]
    got = oracle.confidence(x, sp)
    assert np.allclose(got, want, rtol=1e-12)
    assert np.allclose(oracle.confidence(x + 123.0, sp), got, rtol=1e-10)          # softmax is shift invariant
    assert np.allclose(oracle.confidence(x[:, ::-1], sp), got, rtol=1e-12)         # and permutation invariant
