"""Pins for the oracle's GA (readings G0-G5): operator statistics with closed forms, invariants, a step-by-step
re-derivation on a tiny population, and a brute-force optimum (pin P11 / GA pin v)."""
import numpy as np

from helpers import oracle_lines
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

NP = 9


def _cfg(pop, gens=10, **kw):
    return W.ga_config(pop, gens, **kw)


def test_init_follows_G2_and_is_uniform():
    g = orc.ga_init(3, 16, seed=77, pixel_base=5)
    assert g.dtype == np.float32 and g.min() >= 0.0 and g.max() < 1.0
    for n, i, j in [(0, 0, 0), (1, 3, 5), (2, 15, 8), (0, 7, 4)]:
        r = orc.philox(77, 5 + n, 0, i, j // 4)
        assert g[n, i, j] == np.float32((int(r[j % 4]) >> 8) / 2 ** 24)
    big = orc.ga_init(64, 128, seed=1).astype(np.float64)
    assert abs(big.mean() - 0.5) < 3e-3 and abs(big.var() - 1 / 12) < 2e-3
    assert np.max(np.abs(np.corrcoef(big.reshape(-1, NP).T) - np.eye(NP))) < 0.05


def test_elite_and_pure_selection_distribution():
    pop, k, N = 16, 3, 400
    cfg = _cfg(pop, tournament_k=k, p_cross=0.0, p_mut=0.0)
    rng = np.random.default_rng(0)
    genes = rng.random((N, pop, NP)).astype(np.float32)
    chi2v = rng.random((N, pop)) + 1.0
    out = orc.ga_step(genes, chi2v, 1, cfg, seed=9)
    counts = np.zeros(pop)
    for n in range(N):
        order = np.argsort(chi2v[n], kind="stable")
        rank_of = np.empty(pop, dtype=int); rank_of[order] = np.arange(pop)
        assert np.array_equal(out[n, 0], genes[n, order[0]])                       # elitism
        for i in range(1, pop):
            src = np.where((genes[n] == out[n, i]).all(axis=1))[0]
            assert src.size == 1                                                    # child is a copy of one parent
            counts[rank_of[src[0]]] += 1
    r = np.arange(pop)
    prob = ((pop - r) ** k - (pop - r - 1) ** k) / pop ** k                         # P(winner has rank r), k draws with replacement
    total = counts.sum()
    chisq = ((counts - total * prob) ** 2 / (total * prob + 1e-12))[prob * total > 5].sum()
    assert chisq < 45.0                                                             # ~15 dof, far tail


def test_tie_break_lowest_index():
    pop = 8
    cfg = _cfg(pop, p_cross=0.0, p_mut=0.0)
    genes = np.arange(pop, dtype=np.float32)[None, :, None].repeat(NP, axis=2) / 10
    out = orc.ga_step(genes, np.ones((1, pop)), 1, cfg, seed=4)
    assert np.array_equal(out[0, 0], genes[0, 0])
    # with all chi2 equal every tournament is won by its lowest-index candidate: P(min of 3 uniform draws = m)
    N = 500
    out = orc.ga_step(np.repeat(genes, N, axis=0), np.ones((N, pop)), 1, cfg, seed=4)
    idx = np.rint(out[:, 1:, 0] * 10).astype(int).ravel()
    m = np.arange(pop)
    prob = ((pop - m) ** 3 - (pop - m - 1) ** 3) / pop ** 3
    freq = np.bincount(idx, minlength=pop) / idx.size
    assert np.max(np.abs(freq - prob)) < 0.02


def test_arithmetic_crossover_segment_and_alpha():
    pop, N = 2, 3000
    cfg = _cfg(pop, tournament_k=1, p_cross=1.0, p_mut=0.0)
    genes = np.zeros((N, pop, NP), dtype=np.float32); genes[:, 1, :] = np.linspace(0.2, 1.0, NP, dtype=np.float32)
    out = orc.ga_step(genes, np.tile([1.0, 2.0], (N, 1)), 1, cfg, seed=123)[:, 1, :].astype(np.float64)
    ratio = out / np.linspace(0.2, 1.0, NP)
    # child = B + alpha (A - B) with one alpha for all genes; parents are (0, x): ratio is 0, alpha, 1 - alpha or 1
    assert np.max(ratio.max(axis=1) - ratio.min(axis=1)) < 1e-6
    mixed = ratio[:, 0][(ratio[:, 0] > 1e-9) & (ratio[:, 0] < 1 - 1e-9)]
    assert 0.4 * N < mixed.size < 0.6 * N                       # A != B half of the time
    assert abs(mixed.mean() - 0.5) < 0.03 and abs(mixed.var() - 1 / 12) < 0.01
    # p_cross as a probability
    cfg = _cfg(pop, tournament_k=1, p_cross=0.3, p_mut=0.0)
    out = orc.ga_step(genes, np.tile([1.0, 2.0], (N, 1)), 1, cfg, seed=5)[:, 1, 0].astype(np.float64) / 0.2
    crossed = ((out > 1e-9) & (out < 1 - 1e-9)).mean()
    assert abs(crossed - 0.3 * 0.5) < 0.03


def test_mutation_rate_law_and_bounds():
    pop, N, G = 4, 3000, 10
    cfg = _cfg(pop, gens=G, p_cross=0.0, p_mut=0.25)
    genes = np.full((N, pop, NP), 0.5, dtype=np.float32)
    for t in (1, G):
        s_t = float(cfg["mut_scale"][t])
        d = orc.ga_step(genes, np.ones((N, pop)), t, cfg, seed=31)[:, 1:, :].astype(np.float64) - 0.5
        hit = d != 0
        assert abs(hit.mean() - 0.25) < 0.01
        assert np.max(np.abs(d)) <= s_t * (1 + 1e-6)
        assert abs(d[hit].mean()) < 0.03 * s_t and abs(d[hit].var() - s_t ** 2 / 3) < 0.05 * s_t ** 2
        assert np.allclose(hit.mean(axis=(0, 1)), 0.25, atol=0.03)               # every gene gets its own pair of draws
    assert abs(cfg["mut_scale"][0] - 0.5) < 1e-7 and abs(cfg["mut_scale"][G] - 0.0025) < 1e-9
    # bounds: non-periodic genes clamp to [0,1]; the periodic gene (azimuth, index 2) wraps
    genes = np.full((N, pop, NP), 0.01, dtype=np.float32)
    out = orc.ga_step(genes, np.ones((N, pop)), 1, cfg, seed=32)[:, 1:, :]
    assert out.min() >= 0.0 and out.max() <= 1.0
    assert (out[:, :, 0] == 0.0).mean() > 0.05 and (out[:, :, 2] == 0.0).mean() < 0.001
    assert (out[:, :, 2] > 0.6).mean() > 0.05 and (out[:, :, 0] > 0.6).mean() == 0.0


def test_step_by_step_rederivation_tiny():
    # An independent transcription of reading G3 in numpy binary32, drawing from orc.philox (itself KAT-pinned).
    pop, G, seed, base = 6, 5, 2024, 11
    cfg = _cfg(pop, gens=G, tournament_k=3)
    rng = np.random.default_rng(1)
    genes = rng.random((2, pop, NP)).astype(np.float32)
    chi2v = rng.random((2, pop)); chi2v[1, 3] = chi2v[1, 1]
    f32 = np.float32
    u01 = lambda x: f32(int(x) >> 8) * f32(2.0 ** -24)
    below = lambda x: ((int(x) >> 8) * pop) >> 24
    for t in (1, 4):
        got = orc.ga_step(genes, chi2v, t, cfg, seed=seed, pixel_base=base)
        for n in range(2):
            want = np.empty((pop, NP), dtype=f32)
            want[0] = genes[n, int(np.argmin(chi2v[n]))]
            for i in range(1, pop):
                def tour(k):
                    r = orc.philox(seed, base + n, t, i, k)
                    c = [below(r[m]) for m in range(3)]
                    return min(c, key=lambda q: (chi2v[n, q], q))
                A, B = tour(0), tour(1)
                r2 = orc.philox(seed, base + n, t, i, 2)
                for j in range(NP):
                    g = genes[n, A, j]
                    if u01(r2[0]) < f32(cfg["p_cross"]):
                        d = f32(genes[n, A, j] - genes[n, B, j])
                        g = f32(np.float64(u01(r2[1])) * np.float64(d) + np.float64(genes[n, B, j]))   # fma: one rounding
                    r = orc.philox(seed, base + n, t, i, 3 + j // 2)
                    um, ud = u01(r[2 * (j % 2)]), u01(r[2 * (j % 2) + 1])
                    if um < f32(cfg["p_mut"]):
                        step = f32(f32(2.0) * ud - f32(1.0))
                        g = f32(np.float64(cfg["mut_scale"][t]) * np.float64(step) + np.float64(g))
                    g = f32(g - np.floor(g)) if cfg["periodic"][j] else f32(min(max(g, f32(0)), f32(1)))
                    want[i, j] = g
            assert np.array_equal(got[n], want)


def test_determinism_and_keying():
    cfg = _cfg(8)
    rng = np.random.default_rng(2)
    genes = rng.random((4, 8, NP)).astype(np.float32); chi2v = rng.random((4, 8))
    a = orc.ga_step(genes, chi2v, 2, cfg, seed=5)
    assert np.array_equal(a, orc.ga_step(genes, chi2v, 2, cfg, seed=5))
    assert not np.array_equal(a, orc.ga_step(genes, chi2v, 3, cfg, seed=5))
    assert not np.array_equal(a, orc.ga_step(genes, chi2v, 2, cfg, seed=6))
    # keyed by global pixel id: pixel 2 of a base-0 run == pixel 0 of a base-2 run
    b = orc.ga_step(genes[2:3], chi2v[2:3], 2, cfg, seed=5, pixel_base=2)
    assert np.array_equal(a[2], b[0])


def test_decode_linear_and_log():
    cfg = _cfg(4)
    g = np.array([[0.0] * NP, [1.0] * NP, [0.5] * NP], dtype=np.float32)
    p = orc.decode(g, cfg)
    assert np.allclose(p[0], cfg["lo"]) and np.allclose(p[1], cfg["hi"])
    assert abs(p[2, 0] - np.sqrt(10.0 * 3000.0)) < 1e-9 and abs(p[2, 1] - 90.0) < 1e-12


def test_full_inversion_invariants_and_brute_force_optimum():
    c0 = W.config0()
    ln = oracle_lines(c0["lines"], True)
    lam = c0["lam"]
    truth = W.draw_truth(4, seed=33)
    truth[:, 0] = [400, 900, 1500, 2400]; truth[:, 1] = [30, 60, 120, 150]
    obs = orc.synth(truth, lam, ln)                                              # sigma = 0 data
    # (v) all genes but (B, gamma) fixed at the truth via lo == hi, one pixel at a time
    for n in range(4):
        cfg = W.ga_config(48, 60)
        for j in range(2, NP):
            cfg["lo"][j] = cfg["hi"][j] = truth[n, j]
        cfg["log_scale"][0] = 0; cfg["lo"][0], cfg["hi"][0] = 0.0, 3000.0
        res = orc.ga_invert(obs[n:n + 1], lam, ln, cfg, seed=3, pixel_base=n, want_trace=True)
        tr = res["trace"][0]
        assert np.all(np.diff(tr) <= 0) and tr[-1] == res["chi2"][0]             # (iii) best chi2 non-increasing
        assert np.allclose(res["params"][0, 2:], truth[n, 2:])
        # brute force over a (B, gamma) grid of 50 G x 3 deg cells: GA optimum must lie in the cell of the grid minimum
        Bs, gs = np.arange(0, 3001, 50.0), np.arange(0, 181, 3.0)
        P = np.tile(truth[n], (Bs.size * gs.size, 1))
        P[:, 0] = np.repeat(Bs, gs.size); P[:, 1] = np.tile(gs, Bs.size)
        models = orc.synth(P, lam, ln, threads=8)
        c = np.array([orc.chi2(obs[n], m, cfg["stokes_weight"], cfg["sigma"]) for m in models])
        k = int(np.argmin(c))
        assert abs(res["params"][0, 0] - P[k, 0]) <= 50.0 and abs(res["params"][0, 1] - P[k, 1]) <= 3.0
        assert res["chi2"][0] <= c[k] + 1e-12 or res["chi2"][0] < 1.0
    # genes of the answer decode to the answer; masked pixels give NaN
    cfg = W.ga_config(16, 5)
    res = orc.ga_invert(obs, lam, ln, cfg, seed=3, mask=[1, 0, 1, 1])
    assert np.isnan(res["chi2"][1]) and np.all(np.isnan(res["params"][1]))
    assert np.allclose(orc.decode(res["genes"][[0, 2, 3]], cfg), res["params"][[0, 2, 3]])
    # fitness hook == synth + chi2
    genes = orc.ga_init(4, 16, seed=3)
    f = orc.ga_fitness(genes, obs, lam, ln, cfg)
    m = orc.synth(orc.decode(genes[2, 5], cfg), lam, ln)[0]
    assert abs(f[2, 5] - orc.chi2(obs[2], m, cfg["stokes_weight"], cfg["sigma"])) < 1e-9 * f[2, 5]
