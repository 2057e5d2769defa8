"""GPU parity of ga_uncertainty (eq. 26; reading U1 of DESIGN.md) against the oracle.

Tolerance: the GPU evaluates chi2 in FP32 (relative error eps ~ 1e-5, the rounding of the synthesised
profile itself, which no re-association of the sum removes).  A second difference at step h divides that by h^2, the h/2
level by h^2/4, and the Richardson combination (4 D(h/2) - D(h))/3 adds them: every entry of the Hessian carries a noise
nu ~ 20 eps chi2 / h^2 (~ 10 at h = 2^-6, chi2 = 13).  A perturbation dH changes [H^-1]_ii by at most |H^-1| |dH| relative, i.e.
sigma_i by (1/2) M nu / lambda_min(H).  So parameters of a pixel whose Hessian is well conditioned agree with the FP64 oracle
to a per cent or better, and those of an ill-conditioned pixel (eta0 - dlambdaD - a are nearly degenerate) cannot, on any
FP32 implementation.  The test asserts the distribution (median deviation < 1 %, 90 % of the entries within 5 %) over the
entries the data constrain (oracle sigma_u < 0.05 in box units), and for every such entry the bound 1 % + M nu / (2 lambda_min)
computed from the ORACLE's Hessian; it prints how many pixels that bound leaves meaningful.  And the NaN / zero conventions."""
import os

import numpy as np
import pytest

from helpers import make_obs, oracle_lines
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
NTHREADS = max(1, (os.cpu_count() or 1))


@pytest.fixture(scope="module")
def B():
    from paper_1208_0302_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def dev(a, dtype=np.float32):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


EPS_CHI2 = 1e-5          # relative error of a binary32 chi2 (the fused-fitness test measures it)


def _compare(sig_g, sig_o, hess_o, chi2_o, cfg, min_frac):
    span = cfg["hi"] - cfg["lo"]
    act = span > 0
    rel_u = sig_o / np.where(act, span, 1.0)
    rel_u[:, 0] = sig_o[:, 0] / 1000.0                        # log-scaled B: judge on sigma_B / 1 kG
    good = np.isfinite(sig_o) & np.isfinite(sig_g) & (rel_u < 0.05) & (sig_o > 0)
    assert good.mean() > min_frac, good.mean()
    dev_ = np.abs(sig_g / np.where(sig_o > 0, sig_o, 1.0) - 1.0)
    assert np.median(dev_[good]) < 0.01 and np.quantile(dev_[good], 0.9) < 0.05, (np.median(dev_[good]), np.quantile(dev_[good], 0.9))
    # the worst entries: bounded pixel by pixel by the predicted effect of the FP32 noise on the inverse
    h, M = orc.uncertainty_step(), int(act.sum())
    tight = 0
    for n in np.flatnonzero(good.any(axis=1)):
        lam_min = np.linalg.eigvalsh(hess_o[n][np.ix_(act, act)]).min()
        nu = 20.0 * EPS_CHI2 * chi2_o[n] / h ** 2
        bound = 0.01 + 0.5 * M * nu / lam_min if lam_min > 0 else np.inf
        tight += bound < 0.1
        assert np.all(dev_[n][good[n]] <= bound), (n, dev_[n][good[n]].max(), bound, lam_min)
    print("uncertainty parity: %d pixels compared, %d with a predicted bound below 10 %%; worst deviation %.3g"
          % (good.any(axis=1).sum(), tight, dev_[good].max()))
    return good


@pytest.mark.parametrize("which", ["config0", "config1"])
def test_uncertainty_vs_oracle_at_the_ga_optimum(B, which):
    c = W.config0() if which == "config0" else W.config1()
    N = 48
    truth = W.draw_truth(N, seed=5)
    truth[:, 0] = np.maximum(truth[:, 0], 600.0)               # strong fields: every magnetic parameter is constrained
    mu = np.linspace(0.4, 1.0, N)
    truth, obs, ln = make_obs(c, N, mu=mu, truth=truth, threads=NTHREADS)
    ld = B.line_data_from_workload(c["lines"], True)
    # the optimum both sides differentiate at is the ORACLE's GA optimum, rounded to binary32 (the params array is f32);
    # no output of the CUDA path is ever an oracle input
    res = orc.ga_invert(obs, c["lam"], ln, c["ga"], seed=W.SEED_GA, mu=mu, threads=NTHREADS)
    p32 = res["params"].astype(np.float32)
    sg, cg = B.ga_uncertainty(dev(obs), dev(p32), c["lam"], ld, c["ga"], mu=dev(mu))
    torch.cuda.synchronize()
    # the library's GA returns a chi2 that its own evaluator reproduces at the returned parameters
    gp, gc = B.ga_invert(dev(obs), c["lam"], ld, c["ga"], W.SEED_GA, mu=dev(mu))
    _, cg2 = B.ga_uncertainty(dev(obs), gp, c["lam"], ld, c["ga"], mu=dev(mu))
    assert float(((cg2 - gc).abs() / gc).max()) < 1e-5
    p64 = p32.astype(np.float64)
    so, co, ho = orc.uncertainty(obs, p64, c["lam"], ln, c["ga"], mu=mu, threads=NTHREADS, want_hessian=True)
    assert np.max(np.abs(cg.cpu().numpy() - co) / co) < 2e-4
    sg = sg.cpu().numpy().astype(np.float64)
    # A GA that stopped short of the minimum (config0 is not converged, SURVEY.md par. 7) leaves many pixels on a slope
    # where the full Hessian is indefinite: eq. 26 then has no answer and BOTH sides say NaN for the pixel.
    fin_g, fin_o = np.isfinite(sg).all(axis=1), np.isfinite(so).all(axis=1)
    assert np.mean(fin_g == fin_o) > 0.9, (fin_g.mean(), fin_o.mean())
    print("%s: eq. 26 has an answer (positive definite Hessian) for %d of %d pixels at the GA optimum in FP64, %d on the GPU"
          % (which, fin_o.sum(), N, fin_g.sum()))
    _compare(sg, so, ho, co, c["ga"], 0.08)
    # at the generating truth (the neighbourhood of the true minimum at this noise level) the Hessian is positive
    # definite for nearly every pixel and the well-constrained parameters agree
    t32 = truth.astype(np.float32)
    sg2, _ = B.ga_uncertainty(dev(obs), dev(t32), c["lam"], ld, c["ga"], mu=dev(mu))
    so2, co2, ho2 = orc.uncertainty(obs, t32.astype(np.float64), c["lam"], ln, c["ga"], mu=mu, threads=NTHREADS, want_hessian=True)
    sg2 = sg2.cpu().numpy().astype(np.float64)
    assert np.mean(np.isfinite(so2).all(axis=1)) > 0.8 and np.mean(np.isfinite(sg2).all(axis=1) == np.isfinite(so2).all(axis=1)) > 0.9
    good = _compare(sg2, so2, ho2, co2, c["ga"], 0.4)
    assert good[:, [0, 1, 2, 6]].mean() > 0.7                  # B, gamma, chi, v_los of strong-field pixels


def test_uncertainty_conventions_and_model11(B):
    # fixed genes -> sigma = 0 and left out of H; masked pixels -> NaN; 11-parameter model; prologue weights
    c1 = W.config1()
    lines, lam = c1["lines"], W.grid(6302.0, 96, 0.032)
    ln = oracle_lines(lines, True)
    nm = orc.synth(W.NM_PARAMS[None, :], lam, ln)[0, 0].astype(np.float32)
    ld = B.line_data_from_workload(lines, True, n_params=11, nm_profile=dev(nm))
    N = 24
    truth = W.draw_truth(N, seed=8, npar=11)
    truth[:, 0] = np.maximum(truth[:, 0], 900.0); truth[:, 9] = np.maximum(truth[:, 9], 0.5)
    clean = orc.synth(truth, lam, ln, nm_profile=nm.astype(np.float64), threads=NTHREADS)
    obs = (clean + W.draw_noise(clean.shape, 1e-3)).astype(np.float32).astype(np.float64)
    ga = W.ga_config(64, 1, npar=11, prologue=1)
    ga["lo"][5] = ga["hi"][5] = 0.25                            # damping fixed
    truth[:, 5] = 0.25
    mask = np.ones(N, dtype=np.uint8); mask[::5] = 0
    p32 = truth.astype(np.float32)
    sg, cg = B.ga_uncertainty(dev(obs), dev(p32), lam, ld, ga, mask=dev(mask, np.uint8))
    sg = sg.cpu().numpy().astype(np.float64)
    on = mask.astype(bool)
    assert np.isnan(sg[~on]).all() and np.isnan(cg.cpu().numpy()[~on]).all()
    assert np.all(sg[on, 5] == 0.0)
    so, co = orc.uncertainty(obs[on], p32[on].astype(np.float64), lam, ln, ga, nm_profile=nm.astype(np.float64), threads=NTHREADS)
    assert np.all(so[:, 5] == 0.0)
    assert np.max(np.abs(cg.cpu().numpy()[on] - co) / co) < 2e-4
    # alpha, s, S0 and S1 are nearly degenerate in this model (reading F13), so with noise the full Hessian is
    # indefinite for most pixels: both sides must then say NaN; where it is definite the constrained entries agree
    fin_g, fin_o = np.isfinite(sg[on]).all(axis=1), np.isfinite(so).all(axis=1)
    assert np.mean(fin_g == fin_o) > 0.85, (fin_g.mean(), fin_o.mean())
    # with alpha and s fixed as well the Hessian is the 9-parameter one: definite, and parity is checked on it
    ga2 = dict(ga, lo=ga["lo"].copy(), hi=ga["hi"].copy())
    ga2["lo"][9] = ga2["hi"][9] = 0.75; ga2["lo"][10] = ga2["hi"][10] = 0.1
    t2 = truth.copy(); t2[:, 9] = 0.75; t2[:, 10] = 0.1
    clean2 = orc.synth(t2, lam, ln, nm_profile=nm.astype(np.float64), threads=NTHREADS)
    obs2 = (clean2 + W.draw_noise(clean2.shape, 1e-3)).astype(np.float32).astype(np.float64)
    s2, _ = B.ga_uncertainty(dev(obs2), dev(t2), lam, ld, ga2)
    o2, c2, h2 = orc.uncertainty(obs2, t2.astype(np.float32).astype(np.float64), lam, ln, ga2, nm_profile=nm.astype(np.float64),
                                 threads=NTHREADS, want_hessian=True)
    s2 = s2.cpu().numpy().astype(np.float64)
    assert np.all(s2[:, [5, 9, 10]] == 0.0) and np.all(o2[:, [5, 9, 10]] == 0.0)
    _compare(s2, o2, h2, c2, ga2, 0.25)
