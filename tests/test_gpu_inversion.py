"""GPU parity of the whole inversion (ga_invert through the C ABI) against the oracle GA with the same Philox streams."""
import os

import numpy as np
import pytest

from helpers import make_obs
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


def _errors(params, truth):
    dchi = np.abs(params[:, 2] - truth[:, 2]) % 180.0
    dchi = np.minimum(dchi, 180.0 - dchi)
    return dict(B=np.abs(params[:, 0] - truth[:, 0]), gamma=np.abs(params[:, 1] - truth[:, 1]), chi=dchi,
                v=np.abs(params[:, 6] - truth[:, 6]))


def _compare(gp, gc, res, truth, min_same):
    """north_star's inversion tolerances + the fraction of pixels that end on the identical optimum."""
    gp, gc = gp.cpu().numpy().astype(np.float64), gc.cpu().numpy().astype(np.float64)
    same = np.abs(gc - res["chi2"]) <= 2e-4 * res["chi2"]
    close = np.all(np.abs(gp - res["params"]) <= 1e-4 * (np.abs(res["params"]) + 1.0), axis=1)
    frac = float(np.mean(same & close))
    med_g, med_o = np.median(gc), np.median(res["chi2"])
    assert abs(med_g - med_o) <= 0.01 * med_o, (med_g, med_o)
    eg, eo = _errors(gp, truth), _errors(res["params"], truth)
    for k in eg:
        a, b = np.median(eg[k]), np.median(eo[k])
        assert abs(a - b) <= 0.05 * b, (k, a, b, frac)
    assert frac >= min_same, frac
    return frac


def test_config0_tiny_full_parity(B):
    c0 = W.config0()
    truth, obs, ln = make_obs(c0, c0["n_pixels"], threads=NTHREADS)
    res = orc.ga_invert(obs, c0["lam"], ln, c0["ga"], seed=W.SEED_GA, threads=NTHREADS)
    ld = B.line_data_from_workload(c0["lines"], True)
    gp, gc = B.ga_invert(dev(obs), c0["lam"], ld, c0["ga"], W.SEED_GA)
    _compare(gp, gc, res, truth, min_same=0.9)
    # chi2 returned is the chi2 of the returned parameters: re-evaluated through the library's own per-pixel evaluator
    # (ga_uncertainty's out_chi2; nothing computed by the CUDA path is ever fed to the oracle)
    _, chk = B.ga_uncertainty(dev(obs), gp, c0["lam"], ld, c0["ga"])
    assert float(((gc - chk).abs() / chk).max()) < 1e-5
    # parameters stay inside the box
    p = gp.cpu().numpy()
    lo, hi = c0["ga"]["lo"], c0["ga"]["hi"]
    assert np.all(p >= lo - 1e-6 * np.abs(lo) - 1e-6) and np.all(p <= hi + 1e-6 * np.abs(hi) + 1e-6)


def test_determinism_sharding_mask_and_mu(B):
    c0 = W.config0()
    N = 48
    mu = np.linspace(0.3, 1.0, N)
    truth, obs, ln = make_obs(c0, N, mu=mu, threads=NTHREADS)
    ld = B.line_data_from_workload(c0["lines"], True)
    d_obs, d_mu = dev(obs), dev(mu)
    a = B.ga_invert(d_obs, c0["lam"], ld, c0["ga"], 99, mu=d_mu)
    b = B.ga_invert(d_obs, c0["lam"], ld, c0["ga"], 99, mu=d_mu)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])                   # same seed twice: bit-identical
    # a shard [16:40) with pixel_id_base = 16 reproduces the full run (keying is by global pixel id)
    s = B.ga_invert(d_obs[16:40].contiguous(), c0["lam"], ld, c0["ga"], 99, mu=d_mu[16:40].contiguous(), pixel_id_base=16)
    assert torch.equal(s[0], a[0][16:40]) and torch.equal(s[1], a[1][16:40])
    # mask: skipped pixels give NaN, the others are unchanged
    mask = np.ones(N, dtype=np.uint8); mask[::3] = 0
    m = B.ga_invert(d_obs, c0["lam"], ld, c0["ga"], 99, mu=d_mu, mask=dev(mask, np.uint8))
    mk = torch.from_numpy(mask.astype(bool)).cuda()
    assert torch.isnan(m[1][~mk]).all() and torch.isnan(m[0][~mk]).all()
    assert torch.equal(m[0][mk], a[0][mk]) and torch.equal(m[1][mk], a[1][mk])
    # different seed: different trajectory
    c = B.ga_invert(d_obs, c0["lam"], ld, c0["ga"], 100, mu=d_mu)
    assert not torch.equal(a[0], c[0])
    # mu enters: oracle parity on this mu-varying set
    res = orc.ga_invert(obs, c0["lam"], ln, c0["ga"], seed=99, mu=mu, threads=NTHREADS)
    same = np.abs(a[1].cpu().numpy() - res["chi2"]) <= 2e-4 * res["chi2"]
    assert same.mean() >= 0.85
    # zero generations: best of the initial population
    cz = W.ga_config(64, 0)
    z = B.ga_invert(d_obs, c0["lam"], ld, cz, 5, mu=d_mu)
    rz = orc.ga_invert(obs, c0["lam"], ln, cz, seed=5, mu=mu, threads=NTHREADS)
    assert np.max(np.abs(z[1].cpu().numpy() - rz["chi2"]) / rz["chi2"]) < 2e-4
    # empty input
    e = B.ga_invert(d_obs[:0].contiguous(), c0["lam"], ld, c0["ga"], 1)
    assert e[0].shape == (0, 9)


def test_ragged_population_and_fixed_genes(B):
    # pop not a multiple of 32, tournament of 2, genes fixed through lo == hi, full Zeeman pattern, L = 37
    lines = [W.FE_6301]
    lam = W.grid(W.FE_6301["lambda0"], 37, 0.03)
    cfgw = dict(lines=lines, triplets=False, lam=lam, sigma=1e-3, b_range=(10.0, 3000.0))
    N = 40
    truth, obs, ln = make_obs(cfgw, N, threads=NTHREADS)
    ga = W.ga_config(100, 30, tournament_k=2)
    for j in (3, 5):
        ga["lo"][j] = ga["hi"][j] = 0.5 * (ga["lo"][j] + ga["hi"][j])
    res = orc.ga_invert(obs, lam, ln, ga, seed=8, threads=NTHREADS)
    ld = B.line_data_from_workload(lines, False)
    gp, gc = B.ga_invert(dev(obs), lam, ld, ga, 8)
    same = np.abs(gc.cpu().numpy() - res["chi2"]) <= 2e-4 * res["chi2"]
    assert same.mean() >= 0.85
    assert abs(np.median(gc.cpu().numpy()) - np.median(res["chi2"])) <= 0.01 * np.median(res["chi2"])
    assert np.allclose(gp.cpu().numpy()[:, [3, 5]], res["params"][:, [3, 5]], rtol=1e-6)


def test_config1_subset_full_parity(B):
    # BASELINE config 1 (two lines, L = 128, pop 128, 100 generations) on a 128-pixel subset the oracle finishes in
    # about two minutes on 8 cores; launched exactly as bench.py launches it (one CTA per pixel, 128 threads).
    c1 = W.config1()
    N = 128
    truth, obs, ln = make_obs(c1, N, threads=NTHREADS)
    res = orc.ga_invert(obs, c1["lam"], ln, c1["ga"], seed=W.SEED_GA, threads=NTHREADS)
    ld = B.line_data_from_workload(c1["lines"], True)
    gp, gc = B.ga_invert(dev(obs), c1["lam"], ld, c1["ga"], W.SEED_GA)
    frac = _compare(gp, gc, res, truth, min_same=0.9)
    # (vi) a converged GA falls at or below the expected chi2 at the truth for most pixels
    expect = 128 * 37.0 / (4 * 128 - 9)
    assert np.mean(gc.cpu().numpy() < 1.5 * expect) > 0.5
    print("config1 subset: identical-optimum fraction", frac)


def test_config1_full_size_sampled_parity(B):
    # BASELINE config 1 at FULL size (256 x 256 = 65 536 pixels, L = 128, pop 128, 100 generations), in the launch
    # configuration bench.py times (one ga_invert call over the whole map).  The oracle cannot invert 65 536 pixels in
    # test time, so (a) sixteen blocks of 8 pixels (first, fourteen interior, ragged last) are inverted by the oracle with
    # the same global pixel ids and compared one by one, and (b) properties that hold at any size are checked on the map.
    # (Round 2: four blocks until the far tiers of the Voigt evaluator were re-derived.  The identical-optimum fraction of
    # the population is 91.6 % on the 1024 pixels of tests/test_gpu_statistical_parity.py (90.5 % before that change); a
    # 32-pixel sample has a binomial standard deviation of 5 % around it and came out at 25 of 32, so the sample was made
    # large enough for the unchanged floor of 0.85 to be a test of the kernel and not of the draw.)
    c1 = W.config1()
    N = c1["n_pixels"]
    truth, obs, ln = make_obs(c1, N, threads=NTHREADS)
    ld = B.line_data_from_workload(c1["lines"], True)
    gp, gc = B.ga_invert(dev(obs), c1["lam"], ld, c1["ga"], W.SEED_GA)
    torch.cuda.synchronize()
    gp, gc = gp.cpu().numpy().astype(np.float64), gc.cpu().numpy().astype(np.float64)
    # (b) whole-map properties
    assert np.all(np.isfinite(gc)) and np.all(np.isfinite(gp))
    lo, hi = c1["ga"]["lo"], c1["ga"]["hi"]
    assert np.all(gp >= lo - 1e-6 * np.abs(lo) - 1e-6) and np.all(gp <= hi + 1e-6 * np.abs(hi) + 1e-6)
    expect = 128 * 37.0 / (4 * 128 - 9)                       # E[chi2] at the truth (reading F11)
    assert np.median(gc) < 1.6 * expect
    assert np.mean(gc < 1.5 * expect) > 0.5
    strong = truth[:, 0] > 1000.0                             # strong fields are well constrained at sigma = 1e-3
    assert np.median(np.abs(gp[strong, 0] - truth[strong, 0]) / truth[strong, 0]) < 0.05
    # (a) sampled pixels against the oracle, same Philox streams (keying by global pixel id)
    same = []
    for start in [0] + [4099 + 4367 * k for k in range(14)] + [N - 8]:
        sl = slice(start, start + 8)
        res = orc.ga_invert(obs[sl], c1["lam"], ln, c1["ga"], seed=W.SEED_GA, pixel_base=start, threads=NTHREADS)
        ok = np.abs(gc[sl] - res["chi2"]) <= 2e-4 * res["chi2"]
        close = np.all(np.abs(gp[sl] - res["params"]) <= 1e-4 * (np.abs(res["params"]) + 1.0), axis=1)
        same += list(ok & close)
        # pixels that left the oracle's trajectory still land within the statistical tolerance
        assert np.all(np.abs(gc[sl] - res["chi2"]) <= 0.25 * res["chi2"])
    assert np.mean(same) >= 0.85, np.mean(same)


def test_config3_fulldisc_shape_sampled_parity(B):
    # BASELINE config 3 (full-disc mask, mu per pixel, 80 % quiet / 20 % active, B box [1, 3500] G, 200 generations)
    # on a 64 x 64 rendition of the 2048 x 2048 map; launched as bench.py --workload config3 launches it (mask + mu).
    # 16 active pixels (quiet and active-region) are inverted by the oracle with the same global ids.
    c3 = W.config3(64)
    mask, mu, truth, active = W.fulldisc_truth(c3["n_side"], c3["radius"])
    N = mask.size
    from helpers import oracle_lines
    ln = oracle_lines(c3["lines"], True)
    clean = orc.synth(truth, c3["lam"], ln, mu=mu, threads=NTHREADS)
    obs = (clean + W.draw_noise(clean.shape, c3["sigma"])).astype(np.float32).astype(np.float64)
    ld = B.line_data_from_workload(c3["lines"], True)
    gp, gc = B.ga_invert(dev(obs), c3["lam"], ld, c3["ga"], W.SEED_GA, mask=dev(mask, np.uint8), mu=dev(mu))
    torch.cuda.synchronize()
    gp, gc = gp.cpu().numpy().astype(np.float64), gc.cpu().numpy().astype(np.float64)
    on = mask.astype(bool)
    assert abs(on.mean() - np.pi / 4 * (1000.0 / 1024.0) ** 2) < 0.02           # ~ pi/4 of the pixels are on the disc
    assert np.isnan(gc[~on]).all() and np.isnan(gp[~on]).all() and np.isfinite(gc[on]).all()
    # active-region pixels (B >= 500 G): field strength recovered
    act = on & active
    assert np.median(np.abs(gp[act, 0] - truth[act, 0]) / truth[act, 0]) < 0.05
    # sampled pixels: 8 quiet + 8 active, oracle with mask/mu and the same pixel ids
    idx = np.concatenate([np.flatnonzero(on & ~active)[::400][:8], np.flatnonzero(act)[::80][:8]])
    from concurrent.futures import ThreadPoolExecutor           # one oracle call per pixel id; ctypes releases the GIL
    with ThreadPoolExecutor(NTHREADS) as ex:
        chi_o = list(ex.map(lambda i: orc.ga_invert(obs[i:i + 1], c3["lam"], ln, c3["ga"], seed=W.SEED_GA, mu=mu[i:i + 1],
                                                    pixel_base=int(i), threads=1)["chi2"][0], idx))
    chi_o = np.array(chi_o)
    assert np.all(np.abs(gc[idx] - chi_o) <= 0.25 * chi_o)
    assert np.mean(np.abs(gc[idx] - chi_o) <= 2e-4 * chi_o) >= 0.75


def test_config3_full_size_sampled_parity(B):
    # BASELINE config 3 at FULL size (2048 x 2048, 3.14 M on-disc pixels, 200 generations) in the launch configuration of
    # `bench.py --workload config3` (one ga_invert call with mask and mu; ~65 s on a B200).  The observation cube is
    # synthesised by me_synth + noise as in bench.py, except for 16 sampled on-disc pixels (8 quiet, 8 active-region),
    # whose observations are the oracle's, so that both sides invert identical inputs under the same global pixel ids.
    from helpers import oracle_lines
    c3 = W.config3()
    mask, mu, truth, active = W.fulldisc_truth(c3["n_side"], c3["radius"])
    N = mask.size
    ln = oracle_lines(c3["lines"], True)
    ld = B.line_data_from_workload(c3["lines"], True)
    on = mask.astype(bool)
    idx = np.concatenate([np.flatnonzero(on & ~active)[::330000][:8], np.flatnonzero(on & active)[::80000][:8]])
    assert idx.size == 16
    d_obs, _ = B.me_synth(dev(truth), c3["lam"], ld, mu=dev(mu))
    gen = torch.Generator(device="cuda"); gen.manual_seed(W.SEED_NOISE)
    for s in range(0, N, 1 << 18):
        o = d_obs[s:s + (1 << 18)]
        o.add_(torch.randn(o.shape, generator=gen, device="cuda", dtype=torch.float32), alpha=float(c3["sigma"]))
    clean = orc.synth(truth[idx], c3["lam"], ln, mu=mu[idx], threads=NTHREADS)
    obs_s = (clean + W.draw_noise(clean.shape, c3["sigma"])).astype(np.float32)
    d_obs[torch.from_numpy(idx).cuda()] = torch.from_numpy(obs_s).cuda()
    gp, gc = B.ga_invert(d_obs, c3["lam"], ld, c3["ga"], W.SEED_GA, mask=dev(mask, np.uint8), mu=dev(mu))
    torch.cuda.synchronize()
    gc_h = gc.cpu().numpy().astype(np.float64)
    gp_h = gp.cpu().numpy().astype(np.float64)
    del d_obs
    # whole-map properties
    assert np.isnan(gc_h[~on]).all() and np.isfinite(gc_h[on]).all() and np.isfinite(gp_h[on]).all()
    assert on.sum() == 3141676 or abs(on.sum() - np.pi * 1e6) < 2e3
    expect = 128 * 37.0 / (4 * 128 - 9)
    assert np.median(gc_h[on]) < 1.3 * expect                  # 200 generations: converged to the noise floor
    act = on & active
    assert np.median(np.abs(gp_h[act, 0] - truth[act, 0]) / truth[act, 0]) < 0.03
    # sampled pixels against the oracle
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(NTHREADS) as ex:
        chi_o = list(ex.map(lambda ki: orc.ga_invert(obs_s[ki[0]:ki[0] + 1].astype(np.float64), c3["lam"], ln, c3["ga"],
                                                     seed=W.SEED_GA, mu=mu[ki[1]:ki[1] + 1], pixel_base=int(ki[1]),
                                                     threads=1)["chi2"][0], list(enumerate(idx))))
    chi_o = np.array(chi_o)
    assert np.all(np.abs(gc_h[idx] - chi_o) <= 0.25 * chi_o)
    assert np.mean(np.abs(gc_h[idx] - chi_o) <= 2e-4 * chi_o) >= 0.75


def test_maximum_sizes(B):
    # the largest population (ME_MAX_POP = 1024 -> 1024-thread CTAs) on the longest grid (ME_MAX_L = 512), two lines,
    # and the largest generation count the ABI accepts (schedule table of ME_MAX_GEN + 1 entries) on a cheap problem
    lines, lam = [W.FE_6301, W.FE_6302], W.grid(6302.0, 512, 0.006)
    cfgw = dict(lines=lines, triplets=True, lam=lam, sigma=1e-3, b_range=(10.0, 3000.0))
    N = 2
    truth, obs, ln = make_obs(cfgw, N, threads=NTHREADS)
    ga = W.ga_config(1024, 2)
    res = orc.ga_invert(obs, lam, ln, ga, seed=4, threads=NTHREADS)
    ld = B.line_data_from_workload(lines, True)
    gp, gc = B.ga_invert(dev(obs), lam, ld, ga, 4)
    assert np.max(np.abs(gc.cpu().numpy() - res["chi2"]) / res["chi2"]) < 2e-4
    assert np.allclose(gp.cpu().numpy(), res["params"], rtol=1e-4, atol=1e-4)
    c0 = W.config0()
    t0, o0, l0 = make_obs(c0, 3, threads=NTHREADS)
    gmax = W.ga_config(8, 1023)
    r0 = orc.ga_invert(o0, c0["lam"], l0, gmax, seed=6, threads=3)
    g0 = B.ga_invert(dev(o0), c0["lam"], B.line_data_from_workload(c0["lines"], True), gmax, 6)
    assert np.max(np.abs(g0[1].cpu().numpy() - r0["chi2"]) / r0["chi2"]) < 0.05      # 1023 generations of trajectory
    # one past the limits is refused, nothing is launched
    for bad in (W.ga_config(1025, 2), W.ga_config(8, 1024)):
        with pytest.raises(B.MeError):
            B.ga_invert(dev(o0), c0["lam"], B.line_data_from_workload(c0["lines"], True), bad, 6)
    with pytest.raises(B.MeError):
        B.me_synth(dev(t0), W.grid(6302.5, 513, 0.01), B.line_data_from_workload(c0["lines"], True))


def test_library_built_mutation_schedule_equals_the_table(B):
    # "geometric schedule, table built on host".  A C caller that leaves ga_cfg.mut_scale_table NULL gets the
    # schedule the library builds from mut_scale0 / mut_scale_end (std::pow in double, rounded to binary32); it must be the
    # table both sides are otherwise handed (workloads.mutation_schedule, reading G3), or GPU and oracle trajectories part.
    # Called through ctypes directly: the binding always passes the table.
    import ctypes as C
    c0 = W.config0()
    N = 24
    truth, obs, ln = make_obs(c0, N, threads=NTHREADS)
    ld = B.line_data_from_workload(c0["lines"], True)
    d_obs = dev(obs)
    lam = np.ascontiguousarray(c0["lam"], dtype=np.float64)
    sig = np.ascontiguousarray(c0["ga"]["sigma"], dtype=np.float32)
    outs = []
    for use_table in (True, False):
        c, keep = B.make_ga_cfg(c0["ga"])
        if not use_table:
            c.mut_scale_table = C.POINTER(C.c_float)()             # NULL
        p = torch.empty((N, 9), dtype=torch.float32, device="cuda")
        x = torch.empty((N,), dtype=torch.float32, device="cuda")
        rc = B.lib().ga_invert(C.c_void_p(d_obs.data_ptr()), C.c_int64(N), C.c_void_p(0), sig.ctypes.data_as(C.POINTER(C.c_float)),
                               lam.ctypes.data_as(C.POINTER(C.c_double)), C.c_int(lam.size), C.byref(ld.c), C.byref(c),
                               C.c_uint64(W.SEED_GA), C.c_void_p(p.data_ptr()), C.c_void_p(x.data_ptr()),
                               C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == 0, rc
        torch.cuda.synchronize()
        outs.append((p.cpu().numpy(), x.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])     # bit-identical
    # and the table path is the oracle's trajectory
    res = orc.ga_invert(obs, c0["lam"], ln, c0["ga"], seed=W.SEED_GA, threads=NTHREADS)
    assert np.mean(np.abs(outs[1][1] - res["chi2"]) <= 2e-4 * res["chi2"]) >= 0.85
