"""Pins for the oracle's Zeeman-pattern helper (P10) and Philox4x32-10 (G0)."""
import os
from fractions import Fraction as Fr

import numpy as np

from oracle import api as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_table1_g_eff():
    # Table 1: 6301.5 g_eff = 1.667, 6302.5 g_eff = 2.500
    gl, gu = orc.lande_g(2, 1, 2), orc.lande_g(2, 2, 2)
    assert abs(gl - 11 / 6) < 1e-15 and abs(gu - 1.5) < 1e-15
    assert round(orc.g_eff(gl, 2, gu, 2), 3) == 1.667
    assert round(orc.g_eff(orc.lande_g(2, 1, 1), 1, orc.lande_g(2, 2, 0), 0), 3) == 2.500


def test_6301_pattern_exact_fractions():
    # four contributions to each of the three Zeeman components -> 12 components.
    sh, we, ki = orc.zeeman_pattern((2, 1, 2), (2, 2, 2))
    assert len(sh) == 12 and [(ki == k).sum() for k in (-1, 0, 1)] == [4, 4, 4]
    want = {1: [(Fr(7, 6), Fr(1, 5)), (Fr(3, 2), Fr(3, 10)), (Fr(11, 6), Fr(3, 10)), (Fr(13, 6), Fr(1, 5))],
            0: [(Fr(-2, 3), Fr(2, 5)), (Fr(-1, 3), Fr(1, 10)), (Fr(1, 3), Fr(1, 10)), (Fr(2, 3), Fr(2, 5))]}
    for kind, lst in want.items():
        got = sorted(zip(sh[ki == kind], we[ki == kind]))
        for (s, w), (fs, fw) in zip(got, sorted(lst)):
            assert abs(s - float(fs)) < 1e-14 and abs(w - float(fw)) < 1e-14
    # sigma_blue mirrors sigma_red
    assert np.allclose(np.sort(-sh[ki == -1]), np.sort(sh[ki == 1]))


def test_6302_is_a_normal_triplet():
    sh, we, ki = orc.zeeman_pattern((2, 1, 1), (2, 2, 0))
    assert sorted(zip(ki, sh, we)) == [(-1, -2.5, 1.0), (0, 0.0, 1.0), (1, 2.5, 1.0)]


def test_centre_of_gravity_identity():
    # For any LS transition: weights sum to 1 per kind, centre of gravity of sigma_red = +g_eff, of pi = 0.
    terms = [((2, 1, 2), (2, 2, 2)), ((2, 1, 1), (2, 2, 0)), ((1, 2, 3), (1, 3, 4)), ((0.5, 1, 1.5), (0.5, 2, 2.5)),
             ((1.5, 2, 3.5), (1.5, 1, 2.5)), ((1, 1, 2), (1, 1, 2)), ((0, 0, 0), (0, 1, 1)), ((2.5, 0, 2.5), (2.5, 1, 3.5))]
    for lo, up in terms:
        sh, we, ki = orc.zeeman_pattern(lo, up)
        ge = orc.g_eff(orc.lande_g(*lo), lo[2], orc.lande_g(*up), up[2])
        for k, cog in ((-1, -ge), (0, 0.0), (1, ge)):
            assert abs(we[ki == k].sum() - 1) < 1e-14
            assert abs((we[ki == k] * sh[ki == k]).sum() - cog) < 1e-13
        n_expected = sum(1 for dM in (-1, 0, 1) for Ml in np.arange(-lo[2], lo[2] + 1) if abs(Ml + dM) <= up[2])
        zero_pi = 1 if (lo[2] == up[2] and float(lo[2]).is_integer()) else 0    # M = 0 -> 0 forbidden when dJ = 0
        assert len(sh) == n_expected - zero_pi


def test_philox_known_answers():
    # Known-answer vectors published with the algorithm (Salmon et al. 2011, Random123 kat_vectors, philox4x32 10 rounds).
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        line = line.split("#")[0].split()
        if not line:
            continue
        v = [int(x, 16) for x in line]
        assert list(orc.philox_raw(v[0:4], v[4:6])) == v[6:10]


def test_philox_bijection_and_uniformity():
    # A counter-based generator is a bijection on counters: no collisions; top-24-bit uniforms have mean 1/2, var 1/12.
    outs = np.array([orc.philox(12345, n, 0, 0, 0) for n in range(4096)])
    assert len({tuple(r) for r in outs}) == 4096
    u = (outs >> 8).astype(np.float64) / 2 ** 24
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005
    # key and each counter word all matter
    base = tuple(orc.philox(1, 2, 3, 4, 5))
    for alt in [(2, 2, 3, 4, 5), (1, 9, 3, 4, 5), (1, 2, 9, 4, 5), (1, 2, 3, 9, 5), (1, 2, 3, 4, 9), (1 + (1 << 32), 2, 3, 4, 5)]:
        assert tuple(orc.philox(*alt)) != base
