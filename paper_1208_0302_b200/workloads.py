"""Seeded synthetic inputs shaped like the paper's SOLIS/VSM workloads (Table 1).

This module serves BOTH the CUDA path (bench.py, tests) and the CPU oracle (tests) and therefore holds
none of the method's arithmetic: only the line table, wavelength grids, prior boxes, random truth vectors,
noise, and the full-disc mask / mu / active-region layout.  Profiles are synthesised by whichever side
consumes these inputs.  All randomness is numpy's Philox bit generator with a documented key per purpose.

Parameter order everywhere: [B (G), gamma (deg), chi (deg), eta0, dlambdaD (mA), a, v_los (km/s), S0, S1].
"""
import numpy as np

NPAR = 9
SEED_TRUTH, SEED_NOISE, SEED_GA = 1, 2, 3

# Table 1: Fe I multiplet 816.  Terms as (S, L, J): 5P2-5D2 and 5P1-5D0.
# `strength` = eta0 multiplier relative to 6302.5 (reading F7: 3.54 at T = 5000 K from Table 1's log gf and chi_e).
FE_6301 = dict(name="Fe I 6301.5", lambda0=6301.5091, g_eff=1.667, lower=(2, 1, 2), upper=(2, 2, 2), strength=3.54)
FE_6302 = dict(name="Fe I 6302.5", lambda0=6302.5017, g_eff=2.500, lower=(2, 1, 1), upper=(2, 2, 0), strength=1.0)
LAMBDA_REF = 6302.5017


def grid(centre, L, step):
    """Reading F9: lambda_j = centre + (j - (L-1)/2) * step  (symmetric, half-integer offsets for even L)."""
    return centre + (np.arange(L, dtype=np.float64) - 0.5 * (L - 1)) * step


# 11-parameter model (reading F13): genes 9, 10 = magnetic fill fraction alpha in [0,1], stray-light fraction s in [0,0.3].
# The fixed unpolarised profile I_fixed is the B = 0 profile of this parameter vector at mu = 1 (a typical quiet-Sun
# atmosphere); whichever side consumes it synthesises it (this module holds no arithmetic of the method).
NM_PARAMS = np.array([0.0, 0.0, 0.0, 12.0, 30.0, 0.2, 0.0, 0.25, 0.75])


def prior_box(b_lo=10.0, b_hi=3000.0, npar=NPAR):
    """GA search box = the config's prior box (reading G1)."""
    lo = np.array([b_lo, 0.0, 0.0, 1.0, 20.0, 0.01, -3.0, 0.1, 0.5, 0.0, 0.0])[:npar]
    hi = np.array([b_hi, 180.0, 180.0, 50.0, 45.0, 0.5, 3.0, 0.4, 1.0, 1.0, 0.3])[:npar]
    log_scale = np.array([1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0], dtype=np.int32)[:npar]
    periodic = np.array([0, 0, 1, 0, 0, 0, 0, 0, 0, 0, 0], dtype=np.int32)[:npar]
    return lo, hi, log_scale, periodic


def mutation_schedule(generations, s0=0.5, s_end=0.0025):
    """Reading G3: s_t = s0 (s_end/s0)^(t/G), tabulated in double and rounded to binary32, t = 0..G.  s0 and s_end are
    the binary32 values the C ABI carries (ga_cfg.mut_scale0 / mut_scale_end), so that the table the library builds itself
    when ga_cfg.mut_scale_table is NULL is this table."""
    s0, s_end = float(np.float32(s0)), float(np.float32(s_end))
    t = np.arange(generations + 1, dtype=np.float64)
    return (s0 * (s_end / s0) ** (t / max(generations, 1))).astype(np.float32)


def ga_config(pop, generations, sigma=1e-3, b_lo=10.0, b_hi=3000.0, tournament_k=3, p_cross=0.8, p_mut=None,
              s0=0.5, s_end=0.0025, stokes_weight=(1.0, 4.0, 4.0, 2.0), npar=NPAR, variant=0, prologue=0):
    lo, hi, log_scale, periodic = prior_box(b_lo, b_hi, npar)
    return dict(pop=int(pop), generations=int(generations), tournament_k=int(tournament_k),
                p_cross=float(np.float32(p_cross)), p_mut=float(np.float32(2.0 / npar if p_mut is None else p_mut)),
                mut_scale=mutation_schedule(generations, s0, s_end), lo=lo, hi=hi, log_scale=log_scale, periodic=periodic,
                stokes_weight=np.asarray(stokes_weight, dtype=np.float64), sigma=np.full(4, float(sigma)),
                variant=int(variant), prologue=int(prologue))


def draw_truth(n, seed=SEED_TRUTH, b_lo=10.0, b_hi=3000.0, stream=0, npar=NPAR):
    """iid prior draws (BASELINE config 0): B log-uniform, the rest uniform, S1 = 1 - S0;
    npar = 11 (config 4) appends alpha U[0,1] and s U[0,0.3] from a separate stream."""
    rng = np.random.Generator(np.random.Philox(key=[seed, stream]))
    u = rng.random((n, NPAR))
    p = np.empty((n, npar))
    if npar == 11:
        u2 = np.random.Generator(np.random.Philox(key=[seed, 1000 + stream])).random((n, 2))
        p[:, 9] = u2[:, 0]
        p[:, 10] = 0.3 * u2[:, 1]
    p[:, 0] = b_lo * (b_hi / b_lo) ** u[:, 0]
    p[:, 1] = 180.0 * u[:, 1]
    p[:, 2] = 180.0 * u[:, 2]
    p[:, 3] = 1.0 + 49.0 * u[:, 3]
    p[:, 4] = 20.0 + 25.0 * u[:, 4]
    p[:, 5] = 0.01 + 0.49 * u[:, 5]
    p[:, 6] = -3.0 + 6.0 * u[:, 6]
    p[:, 7] = 0.1 + 0.3 * u[:, 7]
    p[:, 8] = 1.0 - p[:, 7]
    return p


def draw_noise(shape, sigma, seed=SEED_NOISE, stream=0):
    rng = np.random.Generator(np.random.Philox(key=[seed, stream]))
    return sigma * rng.standard_normal(shape)


def config0():
    """Tiny: 64 px, single Fe I 6302.5 triplet, 50 samples at 24 mA, pop 64, 50 generations."""
    return dict(name="config0_tiny", n_pixels=64, lines=[FE_6302], triplets=True, lam=grid(FE_6302["lambda0"], 50, 0.024),
                ga=ga_config(64, 50), sigma=1e-3, b_range=(10.0, 3000.0))


def config1(n_side=256):
    """256x256 map, Fe I 6301.5 + 6302.5 as effective triplets on one 128-point grid centred at 6302.0 A."""
    return dict(name="config1_map256", n_pixels=n_side * n_side, lines=[FE_6301, FE_6302], triplets=True,
                lam=grid(6302.0, 128, 0.024), ga=ga_config(128, 100), sigma=1e-3, b_range=(10.0, 3000.0))


def config2(P=1_000_000):
    c = config1()
    c.update(name="config2_synth_sweep", n_pixels=P)
    return c


def config4(n_side=512):
    """Stress: 512x512, 11-parameter ME (reading F13), two-line 256-point grid at 12 mA, B log-U[1,500], sigma 3e-3,
    pop 512, 300 generations."""
    return dict(name="config4_stress11", n_pixels=n_side * n_side, lines=[FE_6301, FE_6302], triplets=True,
                lam=grid(6302.0, 256, 0.012), ga=ga_config(512, 300, sigma=3e-3, b_lo=1.0, b_hi=500.0, npar=11),
                sigma=3e-3, b_range=(1.0, 500.0), npar=11)


def config3(n_side=2048, radius=1000.0):
    """Full-disc shaped map: circular mask, mu per pixel, 80 % quiet / 20 % active (64-px Gaussian blobs)."""
    return dict(name="config3_fulldisc", n_side=n_side, radius=radius, lines=[FE_6301, FE_6302], triplets=True,
                lam=grid(6302.0, 128, 0.024), ga=ga_config(128, 200, b_lo=1.0, b_hi=3500.0), sigma=1e-3,
                b_range=(1.0, 3500.0))


def fulldisc_truth(n_side=2048, radius=1000.0, seed=SEED_TRUTH, n_blobs=40, blob_sigma=64.0):
    """mask[n_side^2] (uint8), mu[n_side^2], truth[n_side^2, 9] for config 3 (SURVEY.md §8(d) recipe).

    Off-disc pixels carry a valid dummy truth (the quiet-Sun draw) but mask = 0.  The blob scale is expressed
    relative to a 2048 grid so that reduced n_side keeps the same structure.
    """
    rng = np.random.Generator(np.random.Philox(key=[seed, 3]))
    n = n_side * n_side
    scale = n_side / 2048.0
    R = radius * scale
    yy, xx = np.mgrid[0:n_side, 0:n_side].astype(np.float64)
    cx = cy = 0.5 * (n_side - 1)
    r2 = (xx - cx) ** 2 + (yy - cy) ** 2
    mask = (r2 <= R * R)
    mu = np.sqrt(np.clip(1.0 - r2 / (R * R), 0.0, None))
    mu = np.maximum(mu, 0.05)
    # active-region field: sum of signed Gaussian blobs with centres on the disc
    ang = rng.random(n_blobs) * 2 * np.pi
    rad = np.sqrt(rng.random(n_blobs)) * 0.9 * R
    bx, by = cx + rad * np.cos(ang), cy + rad * np.sin(ang)
    sgn = np.where(rng.random(n_blobs) < 0.5, -1.0, 1.0)
    s = blob_sigma * scale
    field = np.zeros((n_side, n_side))
    nearest = np.zeros((n_side, n_side), dtype=np.int64)
    best = np.full((n_side, n_side), -1.0)
    for k in range(n_blobs):
        g = np.exp(-((xx - bx[k]) ** 2 + (yy - by[k]) ** 2) / (2 * s * s))
        field += sgn[k] * g
        upd = g > best
        nearest[upd] = k
        best[upd] = g[upd]
    absf = np.abs(field)
    thr = np.quantile(absf[mask], 0.8)
    active = mask & (absf >= thr)
    truth = draw_truth(n, seed=seed, b_lo=1.0, b_hi=200.0, stream=4)        # quiet Sun: B log-U[1,200]
    norm = (absf - thr) / max(absf.max() - thr, 1e-30)
    a = active.ravel()
    u = rng.random(n)
    truth[a, 0] = 500.0 + 3000.0 * norm.ravel()[a]
    truth[a, 1] = np.where(field.ravel()[a] > 0, 30.0, 150.0) + (40.0 * u[a] - 20.0)
    radial = np.degrees(np.arctan2(yy - by[nearest], xx - bx[nearest])) % 180.0
    truth[a, 2] = radial.ravel()[a]
    return mask.ravel().astype(np.uint8), mu.ravel(), truth, active.ravel()
