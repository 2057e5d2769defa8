"""Pins for the oracle's Faddeeva function (pin P4): closed forms, a library routine, an ODE invariant."""
import math

import numpy as np
from scipy import special

from oracle import api as orc


def test_line_centre_closed_form():
    # H(a, 0) = exp(a^2) erfc(a), F(a, 0) = 0
    a = np.array([1e-3, 0.01, 0.05, 0.3, 0.5, 1.0, 2.0, 5.0, 7.0])
    w = orc.faddeeva(1j * a)
    ref = np.array([math.exp(x * x) * math.erfc(x) for x in a])
    assert np.max(np.abs(w.real - ref) / ref) < 1e-13
    assert np.max(np.abs(w.imag)) < 1e-15


def test_small_damping_limits():
    # a -> 0: H -> exp(-v^2), F -> (2/sqrt(pi)) Dawson(v); first-order term in a is O(a), so compare at a = 1e-3 loosely
    # and check the exact relation at a = 1e-3 against w(v + i a) from scipy separately below.
    v = np.linspace(-6, 6, 241) + 0.013      # keep off the trapezoid nodes
    w = orc.faddeeva(v + 1e-3j)
    assert np.max(np.abs(w.imag - 2 / math.sqrt(math.pi) * special.dawsn(v))) < 3e-3
    assert np.max(np.abs(w.real - np.exp(-v * v))) < 2e-3


def test_against_scipy_wofz():
    rng = np.random.default_rng(7)
    a = 10 ** rng.uniform(-2, math.log10(7.0), 100000)
    v = rng.uniform(-80, 80, a.size)
    z = v + 1j * a
    w, ref = orc.faddeeva(z), special.wofz(z)
    assert np.max(np.abs(w - ref) / np.abs(ref)) < 5e-13
    assert np.max(np.abs(w.real - ref.real) / np.abs(ref.real)) < 5e-12
    # on the trapezoid nodes with small damping (worst case for the pole correction)
    z = np.arange(-13, 14) * 0.5 + 0.01j
    assert np.max(np.abs(orc.faddeeva(z) - special.wofz(z)) / np.abs(special.wofz(z))) < 1e-11
    # above the switch Im z = pi/h the correction term is dropped
    z = rng.uniform(-20, 20, 2000) + 1j * rng.uniform(6.0, 12.0, 2000)
    assert np.max(np.abs(orc.faddeeva(z) - special.wofz(z)) / np.abs(special.wofz(z))) < 1e-13


def test_area_normalisation():
    # Integral of H(a, v) dv = sqrt(pi) for every a
    v = np.linspace(-4000, 4000, 1600001)
    for a in (0.01, 0.2, 0.5):
        H = orc.faddeeva(v + 1j * a).real
        area = np.trapezoid(H, v) + 2 * a / math.sqrt(math.pi) / 4000.0     # Lorentz tails beyond +-4000: a/(sqrt(pi) v^2)
        assert abs(area - math.sqrt(math.pi)) < 2e-6


def test_asymptote_and_ode():
    z = np.array([60 + 0.3j, -75 + 0.02j, 40 + 5j])
    w = orc.faddeeva(z)
    lead = 1j / (math.sqrt(math.pi) * z) * (1 + 0.5 / z ** 2 + 0.75 / z ** 4)
    assert np.max(np.abs(w - lead) / np.abs(w)) < 1e-8
    # w'(z) = -2 z w + 2i/sqrt(pi), by central differences
    rng = np.random.default_rng(3)
    z = rng.uniform(-8, 8, 500) + 1j * rng.uniform(0.05, 3, 500)
    h = 1e-5
    num = (orc.faddeeva(z + h) - orc.faddeeva(z - h)) / (2 * h)
    ana = -2 * z * orc.faddeeva(z) + 2j / math.sqrt(math.pi)
    assert np.max(np.abs(num - ana)) < 1e-8
