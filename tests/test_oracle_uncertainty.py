"""Pins for the oracle's uncertainties (eq. 25-26; reading U1 of DESIGN.md): the finite-difference +
Richardson Hessian is exact on polynomial test functions with a closed-form inverse, and on a noiseless profile it equals
the Gauss-Newton Hessian built from an independent numerical Jacobian of the synthesis."""
import numpy as np

from helpers import oracle_lines
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

H_STEP = orc.uncertainty_step()          # reading U1: 2^-6


def _table(f, M, u0):
    return np.array([f(u0 + orc.uncertainty_offsets(M, e, H_STEP)) for e in range(orc.uncertainty_n_eval(M))])


def test_evaluation_list():
    for M in (2, 9, 11):
        ne = orc.uncertainty_n_eval(M)
        assert ne == 1 + 2 * (2 * M + 2 * M * (M - 1))
        offs = np.array([orc.uncertainty_offsets(M, e, H_STEP) for e in range(ne)])
        assert np.all(offs[0] == 0)
        half = (ne - 1) // 2
        assert np.array_equal(offs[1 + half:], 0.5 * offs[1:1 + half])            # second level = h / 2
        assert len({tuple(o) for o in offs}) == ne                                  # no evaluation is repeated
        assert np.all((offs != 0).sum(axis=1)[1:1 + 2 * M] == 1) and np.all((offs != 0).sum(axis=1)[1 + 2 * M:1 + half] == 2)


def test_quadratic_and_quartic_functions_give_the_exact_sigma():
    rng = np.random.default_rng(0)
    for M in (3, 9, 11):
        R = rng.normal(size=(M, M))
        A = R @ R.T + M * np.eye(M)
        u0, c = rng.random(M), 7.5
        quad = lambda u: c + 0.5 * (u - u0) @ A @ (u - u0)
        want = np.sqrt(np.diag(np.linalg.inv(A)) * c / M)                           # eq. 26
        got = orc.uncertainty_from_chi2(_table(quad, M, u0), M, H_STEP)
        assert np.allclose(got, want, rtol=1e-8)
        # cubic and quartic terms do not change the Hessian at u0; one Richardson level removes their h^2 error exactly
        T = rng.normal(size=(M,)) * 50.0
        quart = lambda u: quad(u) + ((u - u0) ** 3) @ T + 300.0 * np.sum((u - u0) ** 4) + 80.0 * (np.sum(u - u0)) ** 4
        got4 = orc.uncertainty_from_chi2(_table(quart, M, u0), M, H_STEP)
        assert np.allclose(got4, want, rtol=1e-7)
        # without Richardson the quartic term would bias the diagonal by 2 h^2 (300 + 80) * 12 / 12: visible at 1e-3
        # a fixed gene is left out of the Hessian (conditional, not marginal, uncertainty) and gets sigma = 0
        act = np.ones(M, dtype=int); act[1] = 0
        keep = np.flatnonzero(act)
        want_c = np.sqrt(np.diag(np.linalg.inv(A[np.ix_(keep, keep)])) * c / M)
        got_c = orc.uncertainty_from_chi2(_table(quad, M, u0), M, H_STEP, active=act)
        assert got_c[1] == 0.0 and np.allclose(got_c[keep], want_c, rtol=1e-8)
    # a flat direction (singular Hessian) or a saddle gives NaN, never a number
    flat = lambda u: 3.0 + (u[0] - 0.5) ** 2
    assert np.all(np.isnan(orc.uncertainty_from_chi2(_table(flat, 3, np.full(3, 0.5)), 3, H_STEP)))
    saddle = lambda u: 3.0 + (u[0] - 0.5) ** 2 - (u[1] - 0.5) ** 2 + (u[2] - 0.5) ** 2
    assert np.all(np.isnan(orc.uncertainty_from_chi2(_table(saddle, 3, np.full(3, 0.5)), 3, H_STEP)))


def test_noiseless_profile_gives_the_gauss_newton_hessian():
    ln = oracle_lines([W.FE_6302])
    lam = W.grid(W.FE_6302["lambda0"], 48, 0.025)
    cfg = W.ga_config(8, 1)
    L, M = lam.size, 9
    truth = W.draw_truth(3, seed=17)
    truth[:, 0] = [1200.0, 2000.0, 800.0]
    truth[:, 1] = [40.0, 120.0, 70.0]
    obs = orc.synth(truth, lam, ln)
    eps = 1e-3
    noisy = obs + W.draw_noise(obs.shape, eps)
    sig, chi = orc.uncertainty(noisy, truth, lam, ln, cfg)
    assert np.all(np.isfinite(sig)) and np.all(sig > 0)
    lo, hi, w2 = cfg["lo"], cfg["hi"], (cfg["stokes_weight"] / cfg["sigma"]) ** 2
    for n in range(3):
        # independent Jacobian: central first differences of the synthesis in the box coordinate u (p = decode(u))
        def prof(u):
            p = lo + (hi - lo) * u
            p[0] = lo[0] * (hi[0] / lo[0]) ** u[0]
            return orc.synth(p[None, :], lam, ln)[0]
        u0 = (truth[n] - lo) / (hi - lo)
        u0[0] = np.log(truth[n, 0] / lo[0]) / np.log(hi[0] / lo[0])
        J = np.empty((M, 4, L))
        for j in range(M):
            d = np.zeros(M); d[j] = 1e-5
            J[j] = (prof(u0 + d) - prof(u0 - d)) / 2e-5
        Hgn = 2.0 / (4 * L - M) * np.einsum("jsl,ksl,s->jk", J, J, w2)              # d2/du2 of eq. 16 at zero residual
        chi_n = orc.chi2(noisy[n], obs[n], cfg["stokes_weight"], cfg["sigma"])
        assert abs(chi[n] - chi_n) < 1e-9 * chi_n
        want_u = np.sqrt(np.diag(np.linalg.inv(Hgn)) * chi_n / M)
        dpdu = hi - lo; dpdu[0] = truth[n, 0] * np.log(hi[0] / lo[0])
        # the residual term of the full Hessian is O(eps) relative to the Gauss-Newton term here
        assert np.allclose(sig[n], want_u * dpdu, rtol=0.12), (n, sig[n] / (want_u * dpdu))
    # sigma scales with the noise level (H is noise-independent to first order, chi2 is quadratic in it)
    sig2, _ = orc.uncertainty(obs + 2.0 * (noisy - obs), truth, lam, ln, cfg)
    assert np.allclose(sig2 / sig, 2.0, rtol=0.1)


def test_returned_hessian_is_the_one_eq_26_inverts():
    # uncertainty(..., want_hessian=True) hands out the Richardson-extrapolated Hessian in box coordinates: eq. 26 applied to
    # it with numpy's inverse reproduces the returned sigmas, it is symmetric, and asking for it changes nothing else
    c0 = W.config0()
    ln = oracle_lines(c0["lines"], True)
    truth = W.draw_truth(6, seed=31)
    truth[:, 0] = np.maximum(truth[:, 0], 900.0)
    obs = orc.synth(truth, c0["lam"], ln) + W.draw_noise((6, 4, c0["lam"].size), 1e-3, stream=9)
    cfg = c0["ga"]
    sig, chi, H = orc.uncertainty(obs, truth, c0["lam"], ln, cfg, threads=6, want_hessian=True)
    sig2, chi2 = orc.uncertainty(obs, truth, c0["lam"], ln, cfg, threads=6)
    assert np.array_equal(np.nan_to_num(sig), np.nan_to_num(sig2)) and np.array_equal(chi, chi2)
    assert H.shape == (6, 9, 9) and np.allclose(H, np.transpose(H, (0, 2, 1)), rtol=0, atol=0)
    lo, hi = np.asarray(cfg["lo"]), np.asarray(cfg["hi"])
    with np.errstate(all="ignore"):                                            # the log is only taken where the gene is log-scaled
        dpdu = np.where(cfg["log_scale"], truth * np.log(hi / lo), hi - lo)
    seen = 0
    for n in range(6):
        if not np.all(np.isfinite(sig[n])):
            continue
        su = np.sqrt(np.diag(np.linalg.inv(H[n])) * chi[n] / 9.0)              # eq. 26
        assert np.allclose(su * np.abs(dpdu[n]), sig[n], rtol=1e-9)
        seen += 1
    assert seen >= 3
