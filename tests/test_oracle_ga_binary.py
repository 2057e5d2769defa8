"""Pins for the oracle's binary-coded GA variant, the paper's own operators (readings V0-V5 of DESIGN.md):
16-bit genotype and eq. 5 decode, Sobol' initial population and restarts,
one-point crossover of the bit string, LSB-biased bit mutation."""
import numpy as np
from scipy.stats import qmc

from helpers import oracle_lines
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

M = 9


def _cfg(pop, gens=8, **kw):
    return W.ga_config(pop, gens, variant=1, **kw)


def _shift(seed, pixel, j):
    return int(orc.philox(seed, pixel, 0, 0xFFFFFFFF, j // 4)[j % 4]) >> 16


def test_sobol_is_the_library_sequence_and_stratified():
    pts = orc.sobol(0, 4096, 11)
    ref = np.floor(qmc.Sobol(d=11, scramble=False, bits=32).random(4096) * 2.0 ** 32).astype(np.uint64)
    assert np.array_equal(pts.astype(np.uint64), ref)                 # Joe-Kuo direction numbers, Gray-code order
    # dimension 0 is the van der Corput sequence in Gray-code order: bit-reversed n ^ (n >> 1)
    for n in (1, 2, 3, 5, 100, 4095):
        g = n ^ (n >> 1)
        assert int(pts[n, 0]) == int(format(g, "032b")[::-1], 2)
    # (0, m, 1)-net in every dimension: the first 2^m points hit every interval of width 2^-m exactly once
    for m in (3, 7, 12):
        cells = (pts[: 2 ** m] >> np.uint32(32 - m)).astype(np.int64)
        for j in range(11):
            assert np.array_equal(np.sort(cells[:, j]), np.arange(2 ** m))
    # random access: a block starting anywhere equals the slice
    assert np.array_equal(orc.sobol(1000, 50, 11), pts[1000:1050])


def test_eq5_decode_of_sixteen_bit_codes():
    cfg = _cfg(8)
    codes = np.zeros((3, M), dtype=np.float32)
    codes[1, :] = 65535.0
    codes[2, :] = 12345.0
    p = orc.decode(codes, cfg)
    assert np.allclose(p[0], np.where(cfg["log_scale"], cfg["lo"], cfg["lo"]), rtol=1e-12)          # k = 0 -> u_j
    assert np.allclose(p[1], cfg["hi"], rtol=1e-7)                                                  # k = 2^N - 1 -> v_j
    g = np.float32(12345.0) / np.float32(65535.0)
    lin = cfg["lo"] + (cfg["hi"] - cfg["lo"]) * float(g)                                            # eq. 5
    assert np.allclose(p[2, 1:], lin[1:], rtol=1e-12)
    assert abs(p[2, 0] - cfg["lo"][0] * (cfg["hi"][0] / cfg["lo"][0]) ** float(g)) < 1e-9 * p[2, 0]  # log-scaled B (reading G1)
    # resolution: one code step moves the parameter by (v - u) / (2^N - 1)
    codes[2, :] = 12346.0
    assert np.allclose((orc.decode(codes, cfg)[2] - p[2])[1:], ((cfg["hi"] - cfg["lo"]) / 65535.0)[1:], rtol=2e-3)


def test_initial_population_is_shifted_sobol():
    seed, base, pop = 99, 7, 32
    g = orc.ga_init(3, pop, seed, pixel_base=base, npar=11, variant=1)
    assert g.shape == (3, pop, 11) and np.all(g == np.rint(g)) and g.min() >= 0 and g.max() <= 65535
    pts = orc.sobol(1, pop, 11) >> np.uint32(16)
    for n in range(3):
        sh = np.array([_shift(seed, base + n, j) for j in range(11)], dtype=np.uint32)
        assert np.array_equal(g[n].astype(np.uint32), pts ^ sh[None, :])
    # a digital shift keeps the net property: points 1..31 (the origin, point 0, is skipped) fall in 31 different cells
    # of width 1/32 in every dimension
    cells = (g[0].astype(np.uint32) >> np.uint32(11)).astype(int)
    for j in range(11):
        assert len(set(cells[:31, j])) == 31
    assert not np.array_equal(g[0], g[1])                              # pixels differ through the shift


def test_one_point_crossover_structure_and_cut_law():
    pop, N = 4, 1500
    cfg = _cfg(pop, tournament_k=1, p_cross=1.0, p_mut=0.0)
    genes = np.zeros((N, pop, M), dtype=np.float32)
    genes[:, 0::2, :] = 0.0          # even members: all bits 0
    genes[:, 1::2, :] = 65535.0      # odd members: all bits 1
    chi2v = np.tile(np.arange(pop, dtype=np.float64) + 1, (N, 1))
    out = orc.ga_step(genes, chi2v, 1, cfg, seed=5).astype(np.uint32)
    assert np.all(out[:, 0] == 0)                                      # elite = member 0
    c1, c2 = out[:, 1], out[:, 2]                                      # the pair (1, 2)
    assert np.all((c1 ^ c2 == 0xFFFF) | ((c1 == c2)))                  # complementary children unless A and B coincide
    mixed = (c1 ^ c2 == 0xFFFF).all(axis=1)
    bits1 = np.unpackbits(c1[mixed].astype(">u2").view(np.uint8).reshape(-1, 2 * M), axis=1)   # MSB first, gene 0 first
    # one-point crossover: the bit string is constant up to the cut and the complement after it
    changes = (np.diff(bits1.astype(int), axis=1) != 0).sum(axis=1)
    assert np.all(changes == 1)
    cut = 1 + np.argmax(np.diff(bits1.astype(int), axis=1) != 0, axis=1)
    assert cut.min() >= 1 and cut.max() <= 16 * M - 1
    quart = np.histogram(cut, bins=[1, 36, 72, 108, 144])[0] / cut.size
    assert np.max(np.abs(quart - 0.25)) < 0.06 and abs(cut.mean() - 8 * M) < 4.0     # uniform on 1 .. 16M-1
    # without crossover the pair copies its parents
    cfg0 = _cfg(pop, tournament_k=1, p_cross=0.0, p_mut=0.0)
    o0 = orc.ga_step(genes, chi2v, 1, cfg0, seed=5).astype(np.uint32)
    assert np.all((o0 == 0) | (o0 == 0xFFFF)) and np.all((o0.min(axis=2) == o0.max(axis=2)))


def test_mutation_flips_less_significant_bits_more_often():
    pop, N = 2, 4000
    cfg = _cfg(pop, tournament_k=1, p_cross=0.0, p_mut=1.0)
    genes = np.zeros((N, pop, M), dtype=np.float32)
    out = orc.ga_step(genes, np.tile([1.0, 2.0], (N, 1)), 1, cfg, seed=11)[:, 1, :].astype(np.uint32)
    flips = np.array([[(out[:, j] >> b) & 1 for b in range(16)] for j in range(M)]).mean(axis=(0, 2))   # per bit, 0 = LSB
    want = (16 - np.arange(16)) / 64.0                                  # reading V5
    assert np.max(np.abs(flips - want)) < 0.012
    assert np.all(np.diff(flips[::3]) < 0)                              # monotone: LSB most, MSB least
    # p_mut is a per-gene probability
    cfg2 = _cfg(pop, tournament_k=1, p_cross=0.0, p_mut=0.25)
    o2 = orc.ga_step(genes, np.tile([1.0, 2.0], (N, 1)), 1, cfg2, seed=11)[:, 1, :]
    # P(gene changed) = p_mut * P(mask != 0); mask = 0 has small probability, bounded by the LSB law
    assert 0.20 < (o2 != 0).mean() < 0.26
    # transcription of one gene from the raw Philox words
    r = orc.philox(11, 0, 1, 1, 3 + 4 // 2)
    xm, xd = int(r[0]), int(r[1])
    assert int(out[0, 4]) == ((xd & 0xFFFF) & (xd >> 16)) >> (xm & 15)


def test_restart_replaces_the_worst_half_with_the_next_sobol_points():
    pop, G = 16, 8                                                      # N_samp = 2: restarts at t = 2, 4, 6
    cfg = _cfg(pop, gens=G, tournament_k=2, p_cross=0.0, p_mut=0.0)
    rng = np.random.default_rng(3)
    genes = np.rint(rng.random((2, pop, M)) * 65535).astype(np.float32)
    chi2v = rng.random((2, pop)) + 1.0
    seed, base = 17, 40
    for t, r in ((2, 1), (4, 2), (6, 3)):
        out = orc.ga_step(genes, chi2v, t, cfg, seed=seed, pixel_base=base)
        for n in range(2):
            sh = np.array([_shift(seed, base + n, j) for j in range(M)], dtype=np.uint32)
            fresh = (orc.sobol(pop + (r - 1) * (pop // 2) + 1, pop // 2, M) >> np.uint32(16)) ^ sh[None, :]
            assert np.array_equal(out[n, pop // 2:].astype(np.uint32), fresh)           # continues the shifted sequence
            order = np.argsort(chi2v[n], kind="stable")
            live = {tuple(genes[n, i]) for i in order[: pop // 2]}
            for i in range(pop // 2):                                                    # bred from the live half only
                assert tuple(out[n, i]) in live
            assert np.array_equal(out[n, 0], genes[n, order[0]])
    # non-restart generations (odd t, and t = G) breed the whole population and insert nothing
    for t in (1, 3, G):
        out = orc.ga_step(genes, chi2v, t, cfg, seed=seed, pixel_base=base)
        for n in range(2):
            everyone = {tuple(x) for x in genes[n]}
            assert all(tuple(x) in everyone for x in out[n])


def test_binary_variant_inversion_converges_and_is_deterministic():
    ln = oracle_lines([W.FE_6302])
    lam = W.grid(W.FE_6302["lambda0"], 40, 0.03)
    truth = W.draw_truth(6, seed=4)
    truth[:, 0] = np.maximum(truth[:, 0], 800.0)
    obs = orc.synth(truth, lam, ln) + W.draw_noise((6, 4, 40), 1e-3)
    cfg = _cfg(64, gens=40)
    a = orc.ga_invert(obs, lam, ln, cfg, seed=3, threads=6, want_trace=True)
    b = orc.ga_invert(obs[2:4], lam, ln, cfg, seed=3, pixel_base=2, threads=1)
    assert np.array_equal(a["params"][2:4], b["params"]) and np.array_equal(a["chi2"][2:4], b["chi2"])   # global keying
    assert np.all(np.diff(a["trace"], axis=1) <= 0)                    # elitism
    assert np.all(a["trace"][:, -1] < a["trace"][:, 0]) and np.median(a["trace"][:, -1]) < 0.2 * np.median(a["trace"][:, 0])
    assert np.all(a["genes"] == np.rint(a["genes"])) and a["genes"].max() <= 65535
    assert np.all(a["params"] >= cfg["lo"] * (1 - 1e-6)) and np.all(a["params"] <= cfg["hi"] * (1 + 1e-6))
    model = orc.synth(a["params"], lam, ln)
    chk = [orc.chi2(o, m, cfg["stokes_weight"], cfg["sigma"]) for o, m in zip(obs, model)]
    assert np.allclose(chk, a["chi2"], rtol=1e-12)


def test_binary_step_transcription_from_raw_philox_words():
    """An independent numpy transcription of readings V2-V5 from raw Philox words (orc.philox is KAT-pinned): which MEMBER
    a tournament draw names — floor(u P) itself outside restart generations (reading V3 = G3), order[floor(u n_live)]
    at a restart (reading V2) — the pair keying, the bit-mask crossover, the LSB-biased mutation and the fresh points."""
    pop, G, seed, base, k = 10, 8, 77, 5, 3                                 # N_samp = 2: t = 2, 4, 6 restart
    cfg = _cfg(pop, gens=G, tournament_k=k)
    rng = np.random.default_rng(8)
    genes = np.rint(rng.random((2, pop, M)) * 65535).astype(np.float32)
    chi2v = rng.random((2, pop)) + 0.5
    chi2v[1, 6] = chi2v[1, 2]                                               # a tie: lower index wins
    f32 = np.float32
    u01 = lambda x: f32(int(x) >> 8) * f32(2.0 ** -24)
    below = lambda x, n: ((int(x) >> 8) * n) >> 24
    for t in (1, 2, 3, 4, G):
        restart = (t % 2 == 0) and t < G
        n_live = pop - pop // 2 if restart else pop
        got = orc.ga_step(genes, chi2v, t, cfg, seed=seed, pixel_base=base).astype(np.uint32)
        for n in range(2):
            order = sorted(range(pop), key=lambda q: (chi2v[n, q], q))
            want = np.empty((pop, M), dtype=np.uint32)
            want[0] = genes[n, order[0]].astype(np.uint32)
            sh = np.array([_shift(seed, base + n, j) for j in range(M)], dtype=np.uint32)
            for i in range(1, pop):
                if i >= n_live:
                    idx = pop + (t // 2 - 1) * (pop // 2) + (i - n_live) + 1
                    want[i] = (orc.sobol(idx, 1, M)[0] >> np.uint32(16)) ^ sh
                    continue
                key = 2 * ((i + 1) // 2) - 1

                def tour(block):
                    r = orc.philox(seed, base + n, t, key, block)
                    cand = [order[below(r[m], n_live)] if restart else below(r[m], pop) for m in range(k)]
                    return min(cand, key=lambda q: (chi2v[n, q], q))
                A, B = tour(0), tour(1)
                r2 = orc.philox(seed, base + n, t, key, 2)
                cross = u01(r2[0]) < f32(cfg["p_cross"])
                cut = 1 + below(r2[1], 16 * M - 1)
                first, second = (A, B) if i & 1 else (B, A)
                for j in range(M):
                    k1, k2 = int(genes[n, first, j]), int(genes[n, second, j])
                    kk = k1
                    if cross:
                        nhead = min(max(cut - 16 * j, 0), 16)
                        mask = (0xFFFF << (16 - nhead)) & 0xFFFF
                        kk = (k1 & mask) | (k2 & ~mask & 0xFFFF)
                    r = orc.philox(seed, base + n, t, i, 3 + j // 2)
                    xm, xd = int(r[2 * (j % 2)]), int(r[2 * (j % 2) + 1])
                    if u01(xm) < f32(cfg["p_mut"]):
                        kk ^= ((xd & 0xFFFF) & (xd >> 16)) >> (xm & 15)
                    want[i, j] = kk
            assert np.array_equal(got[n], want), (t, n)
