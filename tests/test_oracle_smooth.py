"""Pins of the oracle's view-direction smoothness term (Eq. 9-10), -m "not gpu".

The pin is an independent restatement with numpy library routines (matmul, linalg.norm) in float64, plus the
special cases the definition fixes (delta = 0, delta parallel to d, one perturbation, additivity over s)."""
import math

import numpy as np

import oracle
import synth


def _np_G(sc, F, s):
    enc = list(np.asarray(s, dtype=np.float64))
    for j in range(4):
        for c in range(3):
            enc += [math.sin(2 ** j * float(s[c])), math.cos(2 ** j * float(s[c]))]
    x = np.concatenate([np.asarray(F, dtype=np.float64), np.array(enc)])
    W0, b0, W1, b1, W2, b2 = (np.asarray(a, dtype=np.float64) for a in (sc.W0, sc.b0, sc.W1, sc.b1, sc.W2, sc.b2))
    h = np.maximum(W1 @ np.maximum(W0 @ x + b0, 0) + b1, 0)
    return 1.0 / (1.0 + np.exp(-(W2 @ h + b2)))


def _scene():
    return synth.custom_scene(seed=3, bias_amp=0.4)


def test_smoothness_matches_numpy_restatement():
    sc = _scene()
    O = oracle.OracleScene(sc)
    F, d, delta = synth.smoothness_batch(5, 40, 7, sigma=0.2)
    loss, G = oracle.mlp_smoothness(O, F, d, delta, want_G=True)
    for i in range(40):
        g0 = _np_G(sc, F[i], d[i])
        assert np.allclose(G[i, 0], g0, atol=1e-12)
        ref = 0.0
        for j in range(7):
            s = d[i] + delta[i, j]                                  # fp32 add, as specified
            gs = _np_G(sc, F[i], s)
            assert np.allclose(G[i, j + 1], gs, atol=1e-12)
            cosv = float(np.dot(d[i].astype(np.float64), s.astype(np.float64)) /
                         (np.linalg.norm(d[i].astype(np.float64)) * np.linalg.norm(s.astype(np.float64))))
            ref += cosv * float(np.sum((gs - g0) ** 2))
        assert loss[i] == np.float64(loss[i]) and abs(loss[i] - ref) <= 1e-12 + 1e-9 * abs(ref)
    assert loss.min() >= 0.0 and loss.max() > 1e-6                 # cos > 0 for these small perturbations


def test_smoothness_special_cases():
    sc = _scene()
    O = oracle.OracleScene(sc)
    F, d, delta = synth.smoothness_batch(6, 16, 4, sigma=0.1)
    # no perturbation: every term vanishes exactly
    assert np.array_equal(oracle.mlp_smoothness(O, F, d, np.zeros_like(delta)), np.zeros(16))
    # delta parallel to d: S(d, s) = 1 and the term is the plain squared difference of two G evaluations
    par = (0.25 * d)[:, None, :].repeat(4, axis=1).astype(np.float32)
    loss = oracle.mlp_smoothness(O, F, d, par)
    for i in range(16):
        s = d[i] + par[i, 0]
        x0 = np.concatenate([F[i].astype(np.float64), O.encode_dir(d[i])])
        x1 = np.concatenate([F[i].astype(np.float64), O.encode_dir(s)])
        diff2 = float(np.sum((O.mlp(x1) - O.mlp(x0)) ** 2))
        assert abs(loss[i] - 4 * diff2) <= 1e-9 * diff2 + 1e-15      # cos = 1 up to the fp32 rounding of s
    # additivity over the perturbation set
    full = oracle.mlp_smoothness(O, F, d, delta)
    parts = sum(oracle.mlp_smoothness(O, F, d, delta[:, j:j + 1]) for j in range(4))
    assert np.allclose(full, parts, rtol=1e-12, atol=1e-18)
    # a direction-blind network (zero first-layer weights on the 27 encoding inputs) has zero smoothness loss
    sc.W0[:, 7:] = 0.0
    assert np.array_equal(oracle.mlp_smoothness(oracle.OracleScene(sc), F, d, delta), np.zeros(16))
