"""Pins for the oracle's 11-parameter model (reading F13 of DESIGN.md; eq. 19, stray light
PAPER.md:251):  I = (1 - s)[alpha I^M(p) + (1 - alpha) I(p; B = 0) e] + s I_fixed e.

Each pin is a special case with an independent answer: the 9-parameter synthesis (pinned in test_oracle_synth.py), the
B = 0 closed form through scipy's Faddeeva function, the fixed profile itself, and the continuum of eq. 15.
Also pins the GA's gene bookkeeping for M = 11 (Philox block/lane of every gene; readings G2, G3)."""
import numpy as np
from scipy.special import wofz

from helpers import oracle_lines
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

LINES = [W.FE_6301, W.FE_6302]
LAM = W.grid(6302.0, 96, 0.03)


def _nm(ln, lam=LAM):
    return orc.synth(W.NM_PARAMS[None, :], lam, ln)[0, 0]


def test_alpha_one_no_stray_is_the_nine_parameter_model():
    ln = oracle_lines(LINES)
    p = W.draw_truth(20, seed=5, npar=11)
    p[:, 9], p[:, 10] = 1.0, 0.0
    mu = np.linspace(0.2, 1.0, 20)
    a = orc.synth(p, LAM, ln, mu=mu, nm_profile=_nm(ln))
    b = orc.synth(p[:, :9], LAM, ln, mu=mu)
    assert np.array_equal(a, b)


def test_alpha_zero_is_the_field_free_closed_form():
    ln = oracle_lines(LINES)
    p = W.draw_truth(12, seed=6, npar=11)
    p[:, 9], p[:, 10] = 0.0, 0.0
    mu = 0.7
    out = orc.synth(p, LAM, ln, mu=np.full(12, mu), nm_profile=_nm(ln))
    assert np.all(out[:, 1:] == 0.0)
    for k in range(12):
        eta = np.ones_like(LAM)
        for l in LINES:                                           # pin P1: I = S0 + mu S1 / (1 + eta0 sum r_l H / sqrt(pi))
            dld = p[k, 4] * 1e-3 * l["lambda0"] / W.LAMBDA_REF
            v = ((LAM - l["lambda0"]) - l["lambda0"] * p[k, 6] / 299792.458) / dld
            eta += p[k, 3] * l["strength"] * wofz(v + 1j * p[k, 5]).real / np.sqrt(np.pi)
        want = p[k, 7] + mu * p[k, 8] / eta
        assert np.max(np.abs(out[k, 0] - want)) < 1e-12


def test_full_stray_light_returns_the_fixed_profile():
    ln = oracle_lines(LINES)
    nm = _nm(ln)
    p = W.draw_truth(5, seed=7, npar=11)
    p[:, 10] = 1.0
    out = orc.synth(p, LAM, ln, nm_profile=nm)
    assert np.max(np.abs(out[:, 0] - nm[None, :])) < 1e-15 and np.all(out[:, 1:] == 0.0)
    # the fixed profile is a B = 0 profile: unpolarised by construction, continuum S0 + S1 = 1 for NM_PARAMS
    assert abs(nm[0] - 1.0) < 2e-2 and nm.min() < 0.6


def test_polarisation_scales_with_fill_and_stray_and_intensity_is_bilinear():
    ln = oracle_lines(LINES)
    nm = _nm(ln)
    p = W.draw_truth(16, seed=8, npar=11)
    p[:, 0] = np.maximum(p[:, 0], 800.0)
    out = orc.synth(p, LAM, ln, nm_profile=nm)
    mag = orc.synth(p[:, :9], LAM, ln)
    q = p[:, :9].copy(); q[:, 0] = 0.0
    nonmag = orc.synth(q, LAM, ln)
    al, s = p[:, 9][:, None], p[:, 10][:, None]
    for k in (1, 2, 3):
        assert np.max(np.abs(out[:, k] - (1 - s) * al * mag[:, k])) < 1e-15
    want = (1 - s) * (al * mag[:, 0] + (1 - al) * nonmag[:, 0]) + s * nm[None, :]
    assert np.max(np.abs(out[:, 0] - want)) < 1e-15
    # eq. 19: with no stray light the profile is the alpha-weighted mean of magnetic and non-magnetic
    p0 = p.copy(); p0[:, 10] = 0.0
    o0 = orc.synth(p0, LAM, ln, nm_profile=nm)
    lo, hi = np.minimum(mag[:, 0], nonmag[:, 0]), np.maximum(mag[:, 0], nonmag[:, 0])
    assert np.all(o0[:, 0] >= lo - 1e-14) and np.all(o0[:, 0] <= hi + 1e-14)
    # polarisation degree still <= 1 (pin P8) and the continuum is (1-s)(S0 + mu S1) + s I_fixed (eq. 15)
    assert np.all(np.sqrt((out[:, 1:] ** 2).sum(axis=1)) <= out[:, 0] + 1e-12)
    far = W.grid(6302.0, 4, 40.0)                                 # +-60 A: pure continuum
    nmf = _nm(ln, far)
    of = orc.synth(p, far, ln, nm_profile=nmf)
    cont = (1 - p[:, 10]) * (p[:, 7] + p[:, 8]) + p[:, 10] * nmf[0]
    assert np.max(np.abs(of[:, 0, 0] - cont)) < 2e-4


def test_chi2_uses_nu_with_eleven_parameters():
    L = 40
    obs = np.zeros((4, L)); model = np.zeros((4, L)); model[0, 3] = 0.01
    w, sg = np.array([1.0, 4.0, 4.0, 2.0]), np.full(4, 1e-3)
    assert abs(orc.chi2(obs, model, w, sg, M=11) - (0.01 / 1e-3) ** 2 / (4 * L - 11)) < 1e-9      # nu = 4L - M


def test_ga_gene_bookkeeping_with_eleven_genes():
    M, pop = 11, 12
    g = orc.ga_init(2, pop, seed=21, pixel_base=9, npar=M)
    assert g.shape == (2, pop, M)
    for n, i, j in [(0, 0, 0), (1, 3, 8), (0, 11, 9), (1, 5, 10)]:
        r = orc.philox(21, 9 + n, 0, i, j // 4)                   # reading G2: lane j mod 4 of block floor(j / 4)
        assert g[n, i, j] == np.float32((int(r[j % 4]) >> 8) / 2 ** 24)
    # the first nine genes are the nine-gene initial population (same blocks, same lanes)
    assert np.array_equal(g[:, :, :9], orc.ga_init(2, pop, seed=21, pixel_base=9)[:, :, :9])
    # mutation of gene j draws from block 3 + floor(j/2), lanes (2 (j mod 2), 2 (j mod 2) + 1)   (reading G3)
    cfg = W.ga_config(pop, 5, tournament_k=1, p_cross=0.0, p_mut=1.0, npar=M)
    genes = np.full((1, pop, M), 0.5, dtype=np.float32)
    out = orc.ga_step(genes, np.arange(pop, dtype=np.float64)[None, :] + 1.0, 2, cfg, seed=33, pixel_base=4)
    s_t = cfg["mut_scale"][2]
    for i, j in [(1, 0), (2, 9), (7, 10), (11, 8)]:
        r = orc.philox(33, 4, 2, i, 3 + j // 2)
        ud = np.float32((int(r[2 * (j % 2) + 1]) >> 8) / 2 ** 24)
        want = np.float32(np.float32(0.5) + np.float32(s_t) * (np.float32(2.0) * ud - np.float32(1.0)))
        want = want - np.floor(want) if cfg["periodic"][j] else min(max(want, np.float32(0)), np.float32(1))
        assert abs(float(out[0, i, j]) - float(want)) <= 6e-8      # fma vs two roundings
    assert np.array_equal(out[0, 0], genes[0, 0])                 # elitism


def test_eleven_parameter_inversion_improves_and_stays_in_box():
    ln = oracle_lines([W.FE_6302])
    lam = W.grid(W.FE_6302["lambda0"], 40, 0.03)
    nm = orc.synth(W.NM_PARAMS[None, :], lam, ln)[0, 0]
    truth = W.draw_truth(4, seed=9, npar=11)
    truth[:, 0] = 1500.0
    obs = orc.synth(truth, lam, ln, nm_profile=nm) + W.draw_noise((4, 4, 40), 1e-3)
    cfg = W.ga_config(48, 25, npar=11)
    res = orc.ga_invert(obs, lam, ln, cfg, seed=3, nm_profile=nm, threads=4, want_trace=True)
    assert res["params"].shape == (4, 11)
    assert np.all(np.diff(res["trace"], axis=1) <= 0)             # elitism: best chi2 never increases
    assert np.all(res["trace"][:, -1] < 0.7 * res["trace"][:, 0])      # and it does decrease
    assert np.all(res["params"] >= cfg["lo"] - 1e-9) and np.all(res["params"] <= cfg["hi"] + 1e-9)
    # the returned chi2 is the chi2 of the returned parameters with nu = 4L - 11
    model = orc.synth(res["params"], lam, ln, nm_profile=nm)
    chk = [orc.chi2(o, m, cfg["stokes_weight"], cfg["sigma"], M=11) for o, m in zip(obs, model)]
    assert np.allclose(chk, res["chi2"], rtol=1e-12)
