"""Parity of omerf_mlp_smoothness (Eq. 9-10) against the oracle, through the C-ABI (-m gpu).

Tolerance: G is evaluated with 3xTF32 tensor-core products and fast exp, |dG| <= 4e-6 per output
(measured ~5e-7); a loss term sum_s cos * |G_s - G_0|^2 with per-term differences D then carries an error of at
most 2 * sqrt(3 S l) * 4e-6 + 3 S (4e-6)^2, plus fp32 accumulation 1e-6 relative."""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def omerf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2404_09531_b200 as m
    m.load_library()
    return m


def _run(omerf, sc, F, d, delta, want_G=True):
    import torch
    with omerf.scene_create(sc) as h:
        out = omerf.mlp_smoothness(h, torch.from_numpy(F).cuda(), torch.from_numpy(d).cuda(),
                                   torch.from_numpy(delta).cuda(), want_G=want_G)
        torch.cuda.synchronize()
        assert omerf.last_launch_count(h) == 1
    if want_G:
        return out[0].cpu().numpy().astype(np.float64), out[1].cpu().numpy().astype(np.float64)
    return out.cpu().numpy().astype(np.float64)


# sigma 3.0: perturbed directions up to |s| ~ 10, arguments of the encoding far outside [-pi, pi], negative cosines.
# The 4e-6 bar is a statement about |s| = O(1) (unit directions plus perturbations): the 3xTF32 products keep 2^-21 of
# the magnitude of every product, and s itself is a network input, so the error grows in proportion to max |s|.
@pytest.mark.parametrize("n,S,sigma", [(1000, 15, 0.05), (257, 31, 0.2), (33, 40, 0.1), (5, 1, 0.3), (64, 0, 0.1),
                                       (500, 15, 3.0)])
def test_smoothness_parity(omerf, n, S, sigma):
    import oracle
    sc = synth.custom_scene(seed=3, bias_amp=0.4)
    F, d, delta = synth.smoothness_batch(50 + S, n, S, sigma=sigma)
    loss, G = _run(omerf, sc, F, d, delta)
    ref_loss, ref_G = oracle.mlp_smoothness(oracle.OracleScene(sc), F, d, delta, want_G=True)
    assert np.abs(G - ref_G).max() <= 4e-6
    # |w| <= 1, so sum_s |G_s - G_0|^2 bounds sum_s |w_s| |G_s - G_0|^2 (the two agree for small perturbations, where
    # w ~ 1); with large perturbations the cosine can be negative and the loss itself is no bound
    L = ((ref_G[:, 1:] - ref_G[:, :1]) ** 2).sum(axis=(1, 2)) if S else np.zeros(n)
    tol = 2 * np.sqrt(3 * max(S, 1) * L) * 4e-6 + 3 * max(S, 1) * (4e-6) ** 2 + 1e-6 * L
    assert np.all(np.abs(loss - ref_loss) <= tol), float(np.abs(loss - ref_loss).max())
    if S == 0:
        assert np.array_equal(loss, np.zeros(n))


def test_smoothness_zero_perturbation_and_empty_batch(omerf):
    import torch
    sc = synth.make_scene(0)
    F, d, delta = synth.smoothness_batch(1, 100, 15)
    loss = _run(omerf, sc, F, d, np.zeros_like(delta), want_G=False)
    assert np.array_equal(loss, np.zeros(100))                 # identical rows give identical G: every term is 0
    with omerf.scene_create(sc) as h:
        e = torch.empty((0, 7), device="cuda"), torch.empty((0, 3), device="cuda"), torch.empty((0, 15, 3), device="cuda")
        assert omerf.mlp_smoothness(h, *e).numel() == 0
