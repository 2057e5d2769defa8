"""Pins P1-P9, P11 for the oracle's forward synthesis and chi-square (no GPU)."""
import math

import numpy as np
from scipy import special

from helpers import oracle_lines, single_line
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

C_KMS = 299792.458
ZEEMAN = 4.66857e-13
SQPI = math.sqrt(math.pi)


def _draws(n, seed=11):
    return W.draw_truth(n, seed=seed)


def test_P1_zero_field_closed_form_two_lines():
    cfg = W.config1()
    ln = oracle_lines(cfg["lines"], True)
    lam = cfg["lam"]
    for p, mu in zip(_draws(20), np.linspace(0.1, 1.0, 20)):
        p = p.copy(); p[0] = 0.0
        out = orc.synth(p, lam, ln, mu=[mu])[0]
        assert np.max(np.abs(out[1:])) == 0.0
        den = np.ones_like(lam)
        for l in cfg["lines"]:
            dld = p[4] * 1e-3 * l["lambda0"] / W.LAMBDA_REF
            v = ((lam - l["lambda0"]) - l["lambda0"] * p[6] / C_KMS) / dld
            den += p[3] * l["strength"] * special.wofz(v + 1j * p[5]).real / SQPI
        assert np.max(np.abs(out[0] - (p[7] + mu * p[8] / den))) < 1e-12


def test_P2_longitudinal_field_closed_form():
    g, lam0 = 2.5, 6302.5017
    ln = single_line(g, lam0)
    lam = W.grid(lam0, 81, 0.012)
    for p in _draws(20, seed=5):
        p = p.copy(); p[1] = 0.0
        out = orc.synth(p, lam, ln, mu=[0.8])[0]
        assert np.max(np.abs(out[1])) < 1e-16 and np.max(np.abs(out[2])) < 1e-16
        dld = p[4] * 1e-3
        v = ((lam - lam0) - lam0 * p[6] / C_KMS) / dld
        vB = ZEEMAN * lam0 ** 2 * p[0] / dld
        phi_r = special.wofz(v - g * vB + 1j * p[5]).real / SQPI
        phi_b = special.wofz(v + g * vB + 1j * p[5]).real / SQPI
        assert np.max(np.abs(out[0] + out[3] - (p[7] + 0.8 * p[8] / (1 + p[3] * phi_r)))) < 1e-12
        assert np.max(np.abs(out[0] - out[3] - (p[7] + 0.8 * p[8] / (1 + p[3] * phi_b)))) < 1e-12
    # gamma = 180 deg swaps the roles
    p[1] = 180.0
    out = orc.synth(p, lam, ln, mu=[0.8])[0]
    assert np.max(np.abs(out[0] - out[3] - (p[7] + 0.8 * p[8] / (1 + p[3] * phi_r)))) < 1e-12


def test_P3_closed_form_equals_4x4_solve():
    cfg = W.config1()
    for triplets in (True, False):
        ln = oracle_lines(cfg["lines"], triplets)
        p = _draws(100, seed=2)
        a = orc.synth(p, cfg["lam"], ln, use_solve=False)
        b = orc.synth(p, cfg["lam"], ln, use_solve=True)
        assert np.max(np.abs(a - b)) < 5e-14


def test_P5_angle_symmetries():
    cfg = W.config1()
    ln = oracle_lines(cfg["lines"], False)
    p = _draws(30, seed=9)
    base = orc.synth(p, cfg["lam"], ln)
    q = p.copy(); q[:, 2] += 180.0
    assert np.max(np.abs(orc.synth(q, cfg["lam"], ln) - base)) < 1e-13
    q = p.copy(); q[:, 2] += 90.0
    o = orc.synth(q, cfg["lam"], ln)
    assert np.max(np.abs(o[:, 1:3] + base[:, 1:3])) < 1e-13 and np.max(np.abs(o[:, [0, 3]] - base[:, [0, 3]])) < 1e-13
    q = p.copy(); q[:, 1] = 180.0 - q[:, 1]
    o = orc.synth(q, cfg["lam"], ln)
    assert np.max(np.abs(o[:, 3] + base[:, 3])) < 1e-13 and np.max(np.abs(o[:, 0] - base[:, 0])) < 1e-13
    # Q and U rotate as a spin-2 quantity: chi = 0 -> U = 0 up to magneto-optical terms; Q^2+U^2 invariant under chi
    q = p.copy(); q[:, 2] = 37.0
    o = orc.synth(q, cfg["lam"], ln)
    assert np.max(np.abs((o[:, 1] ** 2 + o[:, 2] ** 2) - (base[:, 1] ** 2 + base[:, 2] ** 2))) < 1e-13


def test_P6_parity_about_line_centre():
    lam0 = 6302.5017
    ln = single_line(2.5, lam0)
    lam = W.grid(lam0, 50, 0.024)
    p = _draws(30, seed=4); p[:, 6] = 0.0
    o = orc.synth(p, lam, ln)
    # differencing lambda - lambda0 near 6302 A leaves ~1e-13 A of asymmetry in the grid itself
    assert np.max(np.abs(o[:, :3] - o[:, :3, ::-1])) < 1e-9
    assert np.max(np.abs(o[:, 3] + o[:, 3, ::-1])) < 1e-9
    assert np.max(np.abs(o[:, 3])) > 1e-3          # not trivially zero


def test_P7_continuum_and_P8_polarisation_degree():
    lam0 = 6302.5017
    ln = single_line(2.5, lam0)
    p = _draws(50, seed=6)
    mu = np.linspace(0.05, 1, 50)
    far = orc.synth(p, np.array([lam0 - 400.0, lam0 + 400.0]), ln, mu=mu)
    cont = p[:, 7] + mu * p[:, 8]                    # eq. 15: I_c = S0 + mu S1
    assert np.max(np.abs(far[:, 0, :] - cont[:, None])) < 2e-6 * 50 and np.max(np.abs(far[:, 1:])) < 1e-6
    cfg = W.config1()
    o = orc.synth(p, cfg["lam"], oracle_lines(cfg["lines"], False), mu=mu)
    pol = np.sqrt((o[:, 1:] ** 2).sum(axis=1))
    assert np.all(pol <= o[:, 0] + 1e-15)
    assert np.all(o[:, 0] > 0) and np.all(o[:, 0] <= cont[:, None] + 1e-12)


def test_P9_weak_field_limit():
    lam0, g = 6302.5017, 2.5
    ln = single_line(g, lam0)
    lam = W.grid(lam0, 101, 0.01)
    h = 1e-3
    for B, tol in ((1.0, 2e-4), (10.0, 2e-3)):
        for p in _draws(10, seed=8):
            p = p.copy(); p[0] = B
            o = orc.synth(p, lam, ln)[0]
            I = lambda d: orc.synth(p, lam + d, ln)[0, 0]
            dI = (8 * (I(h) - I(-h)) - (I(2 * h) - I(-2 * h))) / (12 * h)          # 4th-order central difference
            pred = -g * ZEEMAN * lam0 ** 2 * B * math.cos(math.radians(p[1])) * dI
            scale = np.max(np.abs(pred))
            if scale < 1e-9:
                continue
            assert np.max(np.abs(o[3] - pred)) < tol * scale + 1e-12


def test_anomalous_pattern_reduces_to_triplet_in_weak_field():
    # For B -> 0 the full 6301.5 pattern and its effective triplet give the same Stokes V to first order in B.
    l = dict(W.FE_6301); l["g_eff"] = 5.0 / 3.0
    lam = W.grid(l["lambda0"], 61, 0.02)
    p = _draws(10, seed=12); p[:, 0] = 5.0
    full = orc.synth(p, lam, oracle_lines([l], False, lambda_ref=l["lambda0"]))
    trip = orc.synth(p, lam, oracle_lines([l], True, lambda_ref=l["lambda0"]))
    assert np.max(np.abs(full[:, 3] - trip[:, 3])) < 1e-4 * np.max(np.abs(full[:, 3]))
    assert np.max(np.abs(full[:, 0] - trip[:, 0])) < 1e-5


def test_chi2_definition_and_expectation_at_truth():
    # eq. 16 with nu = 4L - M; reading F11: E[chi2] at the truth = L sum(w^2) / nu
    cfg = W.config0()
    L = cfg["lam"].size
    w, sig = np.array([1.0, 4.0, 4.0, 2.0]), np.full(4, 1e-3)
    rng = np.random.default_rng(0)
    model = rng.random((4, L))
    vals = [orc.chi2(model + 1e-3 * rng.standard_normal((4, L)), model, w, sig) for _ in range(400)]
    expect = L * (w ** 2).sum() / (4 * L - 9)
    assert abs(expect - 9.686) < 1e-3
    assert abs(np.mean(vals) - expect) < 0.03 * expect
    # a single unit residual in Stokes Q at one wavelength contributes (w_Q/sigma)^2 / nu
    obs = model.copy(); obs[1, 7] += 1e-3
    assert abs(orc.chi2(obs, model, w, sig) - 16.0 / (4 * L - 9)) < 1e-9


def test_P11_brute_force_grid_minimum_is_at_truth():
    cfg = W.config0()
    ln = oracle_lines(cfg["lines"], True)
    lam = cfg["lam"]
    w, sig = cfg["ga"]["stokes_weight"], cfg["ga"]["sigma"]
    truth = W.draw_truth(6, seed=21)
    truth[:, 0] = [300, 800, 1200, 1500, 2000, 2500]
    truth[:, 1] = [20, 50, 75, 110, 140, 165]
    for p in truth:
        obs = orc.synth(p, lam, ln)[0]                                  # sigma -> 0 data
        Bs = p[0] + np.linspace(-200, 200, 21)
        gs = p[1] + np.linspace(-15, 15, 21)
        grid = np.array([[b, g] for b in Bs for g in gs])
        P = np.tile(p, (grid.shape[0], 1)); P[:, 0:2] = grid
        models = orc.synth(P, lam, ln, threads=8)
        c = np.array([orc.chi2(obs, m, w, sig) for m in models])
        k = int(np.argmin(c))
        assert abs(grid[k, 0] - p[0]) < 1e-9 and abs(grid[k, 1] - p[1]) < 1e-9 and c[k] < 1e-20


def _profiles_numpy(p, lam, lines):
    """phi_k + i psi_k (k = blue, pi, red) from scipy's wofz: reading F2, written here from SURVEY.md 8(c) steps 1-2."""
    prof = {-1: 0j, 0: 0j, 1: 0j}
    for l in lines:
        dld = p[4] * 1e-3 * l["lambda0"] / l["lambda_ref"]
        v = ((lam - l["lambda0"]) - l["lambda0"] * p[6] / C_KMS) / dld
        vB = ZEEMAN * l["lambda0"] ** 2 * p[0] / dld
        for s, wgt, k in zip(l["shift"], l["weight"], l["kind"]):
            prof[k] = prof[k] + l["strength"] * wgt * special.wofz(v - s * vB + 1j * p[5]) / SQPI
    return prof[-1], prof[0], prof[1]


def test_P12_transverse_field_closed_form_pins_linear_amplitude():
    """gamma = 90 deg, chi = 0: K splits into the (I,Q) block [[eI,eQ],[eQ,eI]] and the (U,V) block, so
    I+Q = S0 + mu S1/(eI+eQ), I-Q = S0 + mu S1/(eI-eQ); the textbook transverse Zeeman effect says light polarised
    ALONG the field sees only the pi component, light polarised ACROSS it the mean of the sigma components:
    eI+eQ = 1 + eta0 phi_p, eI-eQ = 1 + eta0 (phi_b+phi_r)/2 (eq. 8, 12 PAPER.md:185-187, 204-216; reading F1).
    Fixes the factor of the linear-polarisation amplitude kL in oracle/synth.cpp."""
    mu = 0.7
    cases = [([dict(lambda0=6302.5017, strength=1.0, shift=[0.0, -2.5, 2.5], weight=[1, 1, 1], kind=[0, -1, 1],
                    lambda_ref=6302.5017)], W.grid(6302.5017, 81, 0.012))]
    cfg = W.config1()
    two = []
    for l in cfg["lines"]:
        g = l["g_eff"]
        two.append(dict(lambda0=l["lambda0"], strength=l["strength"], shift=[0.0, -g, g], weight=[1, 1, 1],
                        kind=[0, -1, 1], lambda_ref=W.LAMBDA_REF))
    cases.append((two, cfg["lam"]))
    for lines, lam in cases:
        ln = orc.Lines([{k: v for k, v in l.items() if k != "lambda_ref"} for l in lines], lines[0]["lambda_ref"])
        for p in _draws(12, seed=31):
            p = p.copy(); p[1] = 90.0; p[2] = 0.0
            out = orc.synth(p, lam, ln, mu=[mu])[0]
            pb, pp, pr = _profiles_numpy(p, lam, lines)
            Ipar = p[7] + mu * p[8] / (1.0 + p[3] * pp.real)
            Iperp = p[7] + mu * p[8] / (1.0 + p[3] * 0.5 * (pb.real + pr.real))
            assert np.max(np.abs(out[0] + out[1] - Ipar)) < 1e-12
            assert np.max(np.abs(out[0] - out[1] - Iperp)) < 1e-12
            # U and V vanish up to cos(90 deg) = 6e-17 in double
            assert np.max(np.abs(out[2])) < 1e-15 and np.max(np.abs(out[3])) < 1e-15
            assert np.max(np.abs(out[1])) > 1e-4                  # not trivially satisfied


def test_P13_weak_line_expansion_pins_magneto_optical_signs():
    """eta0 -> 0: K = 1 + eta0 A (eq. 8) gives K^-1 e = e - eta0 A e + eta0^2 A^2 e - ...  The first-order term holds only
    the absorption profiles (phi); the magneto-optical profiles (psi = Im w / sqrt(pi), reading F3) enter FIRST at second
    order, e.g. at chi = 0: (A^2 e)_U = aQ' rV' ... = rQ aV - rV aQ.  A is built here in numpy from the matrix of SURVEY.md
    8(c) step 5 (the LL04 form the paper cites) with scipy's wofz; the oracle's profile is compared order by
    order.  Fixes the sign with which Im(kL), Im(kV) enter rho_Q, rho_U, rho_V in oracle/synth.cpp and the sign convention
    of K in stokes_by_solve / stokes_closed_form (eq. 12-13)."""
    lam0, g = 6302.5017, 2.5
    lines = [dict(lambda0=lam0, strength=1.0, shift=[0.0, -g, g], weight=[1, 1, 1], kind=[0, -1, 1], lambda_ref=lam0)]
    ln = single_line(g, lam0)
    lam = W.grid(lam0, 61, 0.015)
    eta0, mu = 1e-4, 0.9
    seen_u = 0
    for p, chi in zip(_draws(12, seed=41), [0.0, 0.0, 0.0, 0.0, 20.0, 65.0, 100.0, 140.0, 0.0, 33.0, 90.0, 170.0]):
        p = p.copy(); p[0] = max(p[0], 600.0); p[2] = chi; p[3] = eta0
        p[1] = min(max(p[1], 25.0), 155.0)
        if abs(p[1] - 90.0) < 10.0:
            p[1] = 60.0                                           # keep both eta_V and eta_Q away from zero
        out = orc.synth(p, lam, ln, mu=[mu])[0]
        x = out / (mu * p[8]); x[0] -= p[7] / (mu * p[8])         # K^-1 e
        pb, pp, pr = _profiles_numpy(p, lam, lines)
        gam, ch = math.radians(p[1]), math.radians(p[2])
        s2, c2 = math.sin(gam) ** 2, math.cos(gam) ** 2
        kI = 0.5 * (pp * s2 + 0.5 * (pb + pr) * (1 + c2))
        kL = 0.5 * (pp - 0.5 * (pb + pr)) * s2
        kV = 0.5 * (pr - pb) * math.cos(gam)
        aI, aQ, aU, aV = kI.real, kL.real * math.cos(2 * ch), kL.real * math.sin(2 * ch), kV.real
        rQ, rU, rV = kL.imag * math.cos(2 * ch), kL.imag * math.sin(2 * ch), kV.imag
        for j in range(lam.size):
            A = np.array([[aI[j], aQ[j], aU[j], aV[j]],
                          [aQ[j], aI[j], rV[j], -rU[j]],
                          [aU[j], -rV[j], aI[j], rQ[j]],
                          [aV[j], rU[j], -rQ[j], aI[j]]])
            e = np.array([1.0, 0.0, 0.0, 0.0])
            first, second = -A @ e, A @ A @ e
            got1 = (x[:, j] - e) / eta0
            got2 = (x[:, j] - e - eta0 * first) / eta0 ** 2
            assert np.max(np.abs(got1 - first)) < 3e-4 * np.max(np.abs(A)) + 1e-12
            assert np.max(np.abs(got2 - second)) < 2e-3 * np.max(np.abs(second)) + 1e-7
        if chi == 0.0:
            # the magneto-optical cross term alone: U(chi = 0) = mu S1 eta0^2 (rQ aV - rV aQ), sign included
            U2 = mu * p[8] * eta0 ** 2 * (rQ * aV - rV * aQ)
            big = np.abs(U2) > 0.2 * np.max(np.abs(U2))
            assert np.max(np.abs(U2)) > 1e-12
            assert np.all(np.sign(out[2][big]) == np.sign(U2[big]))
            assert np.max(np.abs(out[2] - U2)) < 2e-3 * np.max(np.abs(U2))
            seen_u += 1
    assert seen_u >= 4
