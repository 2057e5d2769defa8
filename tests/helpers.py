"""Shared test helpers: oracle-side line lists and observation builders (tests may use oracle/)."""
import numpy as np

from oracle import api as orc
from paper_1208_0302_b200 import workloads as W


def oracle_lines(lines, triplets=True, lambda_ref=W.LAMBDA_REF):
    out = []
    for l in lines:
        if triplets:
            g = l["g_eff"]
            sh, we, ki = [0.0, -g, g], [1.0, 1.0, 1.0], [0, -1, 1]
        else:
            sh, we, ki = orc.zeeman_pattern(l["lower"], l["upper"])
        out.append(dict(lambda0=l["lambda0"], strength=l["strength"], shift=sh, weight=we, kind=ki))
    return orc.Lines(out, lambda_ref)


def single_line(g=2.5, lambda0=6302.5017, strength=1.0):
    return orc.Lines([dict(lambda0=lambda0, strength=strength, shift=[0.0, -g, g], weight=[1, 1, 1], kind=[0, -1, 1])], lambda0)


def make_obs(cfg, n, seed_truth=W.SEED_TRUTH, seed_noise=W.SEED_NOISE, mu=None, truth=None, threads=8):
    """Oracle-synthesised observations: truth[n,9], obs[n,4,L] = synth(truth) + N(0, sigma)."""
    if truth is None:
        truth = W.draw_truth(n, seed=seed_truth, b_lo=cfg["b_range"][0], b_hi=cfg["b_range"][1])
    ln = oracle_lines(cfg["lines"], cfg["triplets"])
    clean = orc.synth(truth, cfg["lam"], ln, mu=mu, threads=threads)
    obs = clean + W.draw_noise(clean.shape, cfg["sigma"], seed=seed_noise)
    obs = obs.astype(np.float32).astype(np.float64)       # the cube is binary32 ([N,4,L] f32): both sides read the same values
    return truth, obs, ln
