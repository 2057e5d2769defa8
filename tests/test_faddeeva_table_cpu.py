"""Host logic behind the device Voigt evaluator: the generated coefficient header (csrc/gen_faddeeva_table.py).

No kernel runs here.  The far tiers of the FP32 evaluator are polynomials in r = 1/|z|^2 whose
coefficients are tabulated polynomials in a^2, obtained by regrouping the asymptotic series of w(z) and truncating its Chebyshev
expansion on [0, 1/T^2].  These tests check that derivation against scipy.special.wofz (a library routine, not the oracle and
not the CUDA path), and that the committed header is what the committed generator writes.
"""
import importlib.util
import math
import os

import numpy as np
import pytest
from scipy.special import wofz

CSRC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_1208_0302_b200", "csrc")


@pytest.fixture(scope="module")
def gen():
    spec = importlib.util.spec_from_file_location("gen_faddeeva_table", os.path.join(CSRC, "gen_faddeeva_table.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_committed_header_is_the_generators_output(gen, tmp_path):
    out = tmp_path / "faddeeva_table.h"
    gen.main(str(out))
    assert out.read_text() == open(os.path.join(CSRC, "faddeeva_table.h")).read()


def test_regrouped_series_is_the_asymptotic_series(gen):
    # H = a r X(r; A), F = v r Y(r; A) with the UN-economised series must reproduce w(z) far out (|z| = 12: the terms fall fast)
    X, Y = gen.far_series(8)
    for a in (0.02, 0.3, 0.75):
        for v in (12.0, 17.5, 40.0):
            r, A = 1.0 / (v * v + a * a), a * a
            x = sum(float(c) * r ** i * A ** p for (i, p), c in X.items()) / math.sqrt(math.pi)
            y = sum(float(c) * r ** i * A ** p for (i, p), c in Y.items()) / math.sqrt(math.pi)
            w = wofz(v + 1j * a)
            assert abs(a * r * x - w.real) < 2e-12 and abs(v * r * y - w.imag) < 2e-12
    # leading coefficients as printed in DESIGN.md / me_device.cuh
    assert X[(1, 0)] == gen.Fraction(3, 2) and X[(2, 0)] == gen.Fraction(15, 4) and X[(2, 1)] == -2 and X[(3, 1)] == -15
    assert Y[(1, 0)] == gen.Fraction(1, 2) and Y[(2, 0)] == gen.Fraction(3, 4) and Y[(2, 1)] == -2 and Y[(3, 1)] == -9


def test_economised_tiers_meet_their_stated_error(gen):
    # the numbers DESIGN.md quotes; in double, i.e. without the FP32 rounding of the device evaluation
    eh, ef = gen.far_error(3, gen.FAR, 14.0)
    assert gen.FAR == 4.5 and eh < 6e-8 and ef < 1.8e-7, (eh, ef)
    eh, ef = gen.far_error(1, gen.FAR_LIN, 80.0)
    assert gen.FAR_LIN == 12.0 and eh < 5e-8 and ef < 2.3e-7, (eh, ef)
    # economisation beats plain truncation of the same series at the same degree (why the tiers could move inwards)
    X, Y = gen.far_series(gen.KFAR)
    a, T = 0.3, gen.FAR
    v = np.linspace(math.sqrt(T * T - a * a), 14.0, 4000)
    r = 1.0 / (v * v + a * a)
    trunc = sum(float(c) * r ** i * (a * a) ** p for (i, p), c in X.items() if i <= 3) / math.sqrt(math.pi)
    assert np.abs(a * r * trunc - wofz(v + 1j * a).real).max() > 5 * gen.far_error(3, T, 14.0)[0]


def test_economisation_matrix_is_a_chebyshev_truncation(gen):
    R = 1.0 / 20.25
    M = gen.economise_matrix(6, 3, R)
    # polynomials of degree <= 3 pass unchanged; r^4 loses exactly its T_4 term, whose size on [0, R] is R^4 / 128
    assert np.allclose(M[:, :4], np.eye(4), atol=1e-12)
    r = np.linspace(0.0, R, 2001)
    err = r ** 4 - sum(M[j, 4] * r ** j for j in range(4))
    assert abs(np.abs(err).max() - R ** 4 / 128.0) < 1e-3 * R ** 4 / 128.0
