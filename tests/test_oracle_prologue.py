"""Pins for the oracle's per-pixel prologue (readings W1, P1 of DESIGN.md): inverse-max weights (eq. 20-23,
PAPER.md:259-270) and the polarity restriction of the inclination."""
import numpy as np

from helpers import oracle_lines, single_line
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W


def test_inverse_max_weights_are_eq_20_to_23():
    rng = np.random.default_rng(0)
    obs = rng.normal(0, 0.01, (5, 4, 33))
    obs[:, 0] = 1.0 - 0.6 * np.exp(-np.linspace(-3, 3, 33) ** 2)[None, :] + rng.normal(0, 1e-3, (5, 33))
    cfg = W.ga_config(8, 2, prologue=1)
    out = orc.prologue(obs, cfg)
    assert np.allclose(out[:, 0], 1.0 / (obs[:, 0].max(axis=1) - obs[:, 0].min(axis=1)), rtol=1e-14)     # eq. 20
    for s in (1, 2, 3):
        assert np.allclose(out[:, s], 1.0 / np.abs(obs[:, s]).max(axis=1), rtol=1e-14)                   # eq. 21-23
    assert np.all(out[:, 4] == cfg["lo"][1]) and np.all(out[:, 5] == cfg["hi"][1])                       # box untouched
    # the weights equalise the four terms: every weighted profile has unit amplitude
    assert np.allclose(np.abs(obs[:, 1:] * out[:, 1:4, None]).max(axis=2), 1.0)
    # an empty Stokes parameter is floored at the noise level instead of dividing by zero
    obs[2, 2] = 0.0
    assert orc.prologue(obs, cfg)[2, 2] == 1.0 / cfg["sigma"][2]
    # bit clear: the configured weights come back
    assert np.allclose(orc.prologue(obs, W.ga_config(8, 2))[:, :4], [1.0, 4.0, 4.0, 2.0])


def test_polarity_follows_the_lobe_order_of_synthetic_profiles():
    # reading F4 (pinned by the weak-field limit, P9): gamma < 90 deg puts the POSITIVE lobe of V on the blue side
    ln = single_line()
    lam = W.grid(6302.5017, 61, 0.02)
    p = W.draw_truth(40, seed=13)
    p[:, 0] = np.maximum(p[:, 0], 300.0)
    p[:, 6] = 0.0
    p[:20, 1] = np.linspace(5, 80, 20)
    p[20:, 1] = np.linspace(100, 175, 20)
    obs = orc.synth(p, lam, ln)
    cfg = W.ga_config(8, 2, prologue=2)
    out = orc.prologue(obs, cfg)
    assert np.all(out[:20, 4] == 0.0) and np.all(out[:20, 5] == 90.0)
    assert np.all(out[20:, 4] == 90.0) and np.all(out[20:, 5] == 180.0)
    assert np.allclose(out[:, :4], [1.0, 4.0, 4.0, 2.0])                                                 # weights untouched
    # a box that is already narrower is only intersected
    cfg2 = dict(cfg, lo=cfg["lo"].copy(), hi=cfg["hi"].copy()); cfg2["lo"][1], cfg2["hi"][1] = 30.0, 120.0
    o2 = orc.prologue(obs, cfg2)
    assert np.all(o2[:20, 4] == 30.0) and np.all(o2[:20, 5] == 90.0) and np.all(o2[20:, 4] == 90.0) and np.all(o2[20:, 5] == 120.0)


def test_inversion_with_prologue_uses_the_per_pixel_weights_and_box():
    ln = oracle_lines([W.FE_6302])
    lam = W.grid(W.FE_6302["lambda0"], 40, 0.03)
    truth = W.draw_truth(6, seed=21)
    truth[:, 0] = np.maximum(truth[:, 0], 1000.0)
    obs = orc.synth(truth, lam, ln) + W.draw_noise((6, 4, 40), 1e-3)
    cfg = W.ga_config(48, 30, prologue=3)
    res = orc.ga_invert(obs, lam, ln, cfg, seed=5, threads=6)
    pro = orc.prologue(obs, cfg)
    # inclination of every pixel inside its polarity box, on the side of the truth for these strong fields
    assert np.all(res["params"][:, 1] >= pro[:, 4] - 1e-9) and np.all(res["params"][:, 1] <= pro[:, 5] + 1e-9)
    assert np.all((res["params"][:, 1] < 90.0) == (truth[:, 1] < 90.0))
    # the returned chi2 is eq. 16 with the per-pixel inverse-max weights
    model = orc.synth(res["params"], lam, ln)
    chk = [orc.chi2(o, m, w[:4], cfg["sigma"]) for o, m, w in zip(obs, model, pro)]
    assert np.allclose(chk, res["chi2"], rtol=1e-12)
    # and differs from the fixed-weight run
    fixed = orc.ga_invert(obs, lam, ln, W.ga_config(48, 30), seed=5, threads=6)
    assert not np.allclose(fixed["chi2"], res["chi2"])
