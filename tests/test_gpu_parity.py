"""GPU parity tests: the CUDA path (through the C ABI via paper_1208_0302_b200.binding) against the CPU oracle,
element by element on the same seeded inputs.  Run on the B200 box: pytest -m gpu.

Tolerances:
  forward synthesis   max |dStokes| / I_c <= 2e-5                      (north_star)
  fused fitness       |dchi2| / chi2 <= 2e-4 (typically 1e-5)          (SURVEY.md par. 7: trajectory parity needs <~ 1e-4)
  GA discrete state   bit-exact given the same fitness                 (readings G0-G3)
  full inversion      median chi2 within 1 %, median |dB|,|dgamma|,|dchi|,|dv| within 5 % of the oracle's (north_star)
"""
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
    assert torch.cuda.is_available()
    return binding


def dev(a, dtype=np.float32):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


# ---------------------------------------------------------------------------------------------------- RNG
def test_philox_device_bit_exact(B):
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")):
        line = line.split("#")[0].split()
        if not line:
            continue
        v = [int(x, 16) for x in line]
        got = B.me_philox(v[4] | (v[5] << 32), *v[0:4])
        assert list(got) == v[6:10]
    n = 20000
    seed = 0x1234567890ABCDEF
    got = B.me_philox_many(seed, 4294967000, 7, 9, 2, n).cpu().numpy().view(np.uint32)   # c0 wraps past 2^32
    for i in list(range(0, 600)) + list(range(n - 200, n)):
        assert tuple(got[i]) == tuple(orc.philox(seed, (4294967000 + i) & 0xffffffff, 7, 9, 2))
    assert len({tuple(r) for r in got}) == n


# ---------------------------------------------------------------------------------------------------- Faddeeva
def test_faddeeva_device_vs_oracle(B):
    rng = np.random.default_rng(5)
    n = 400000
    a = rng.uniform(0.01, 0.5, n).astype(np.float32)
    v = np.concatenate([rng.uniform(-8, 8, n // 2), rng.uniform(-90, 90, n - n // 2)]).astype(np.float32)
    v[:7] = [0.0, 5.5, -5.5, 5.4999, 1e-6, 89.0, -0.5]
    H, F = B.me_faddeeva(dev(v), dev(a))
    H, F = H.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)
    ref = orc.faddeeva(v.astype(np.float64) + 1j * a.astype(np.float64))
    assert np.max(np.abs(H - ref.real)) < 1.5e-6 and np.max(np.abs(F - ref.imag)) < 1.5e-6
    wing = (v.astype(np.float64) ** 2 + a.astype(np.float64) ** 2) >= 5.6 ** 2
    assert np.max(np.abs(H - ref.real)[wing] / ref.real[wing]) < 3e-6      # no cancellation in the wing form
    assert np.max(np.abs(F - ref.imag)[wing] / np.abs(ref.imag[wing])) < 2e-6
    # where H matters for the profiles (H*eta ~ 1): relative accuracy in the core
    core = ~wing & (ref.real > 1e-3)
    assert np.max(np.abs(H - ref.real)[core] / ref.real[core]) < 5e-4


# ---------------------------------------------------------------------------------------------------- synthesis
SYNTH_CASES = [
    ("config0 single triplet L=50", [W.FE_6302], True, W.grid(W.FE_6302["lambda0"], 50, 0.024), 1000 + 7),
    ("config1 two triplets L=128", [W.FE_6301, W.FE_6302], True, W.grid(6302.0, 128, 0.024), 2048 + 5),
    ("full Zeeman patterns L=127 (ragged)", [W.FE_6301, W.FE_6302], False, W.grid(6302.0, 127, 0.024), 517),
    ("single anomalous line L=3", [W.FE_6301], False, W.grid(W.FE_6301["lambda0"], 3, 0.05), 33),
    ("config4-like grid L=256", [W.FE_6301, W.FE_6302], True, W.grid(6302.0, 256, 0.012), 300),
    ("single triplet L=52 (ragged last store chunk of aligned rows)", [W.FE_6302], True, W.grid(W.FE_6302["lambda0"], 52, 0.024), 129),
    ("three lines (run-time line count) L=64", [W.FE_6301, W.FE_6302, dict(W.FE_6302, lambda0=6302.0)], True, W.grid(6302.0, 64, 0.03), 100),
]


@pytest.mark.parametrize("name,lines,triplets,lam,P", SYNTH_CASES, ids=[c[0] for c in SYNTH_CASES])
def test_me_synth_vs_oracle(B, name, lines, triplets, lam, P):
    p = W.draw_truth(P, seed=101)
    mu = np.random.default_rng(1).uniform(0.05, 1.0, P)
    ref = orc.synth(p, lam, oracle_lines(lines, triplets), mu=mu, threads=NTHREADS)
    ld = B.line_data_from_workload(lines, triplets)
    out, _ = B.me_synth(dev(p), lam, ld, mu=dev(mu))
    out = out.cpu().numpy().astype(np.float64)
    cont = (p[:, 7] + mu * p[:, 8])[:, None, None]
    err = np.abs(out - ref) / cont
    print("forward synthesis: max |dStokes| / I_c = %.2e (north_star bound 2e-5)" % err.max())
    assert err.max() <= 2e-5, (name, err.max(), np.unravel_index(err.argmax(), err.shape))
    # mu = NULL means mu = 1
    out1, _ = B.me_synth(dev(p[:64]), lam, ld)
    ref1 = orc.synth(p[:64], lam, oracle_lines(lines, triplets), threads=NTHREADS)
    assert np.max(np.abs(out1.cpu().numpy() - ref1) / (p[:64, 7] + p[:64, 8])[:, None, None]) <= 2e-5


def test_me_synth_extremes_and_chi2(B):
    c1 = W.config1()
    lam = c1["lam"]
    lo, hi, _, _ = W.prior_box(1.0, 3500.0)
    rng = np.random.default_rng(3)
    corners = np.where(rng.random((512, 9)) < 0.5, lo, hi)        # corners of the search box
    corners[:, 0] = np.where(rng.random(512) < 0.3, 0.0, corners[:, 0])   # and B = 0
    ref = orc.synth(corners, lam, oracle_lines(c1["lines"], True), threads=NTHREADS)
    ld = B.line_data_from_workload(c1["lines"], True)
    out, _ = B.me_synth(dev(corners), lam, ld)
    err = np.abs(out.cpu().numpy() - ref) / (corners[:, 7] + corners[:, 8])[:, None, None]
    print("forward synthesis: max |dStokes| / I_c = %.2e (north_star bound 2e-5)" % err.max())
    assert err.max() <= 2e-5
    zero_b = corners[:, 0] == 0.0
    assert float(out[torch.from_numpy(zero_b).cuda()][:, 1:].abs().max()) == 0.0     # B = 0 => Q = U = V = 0 exactly
    # fused chi2 against a fixed profile (config 2), with and without the Stokes output
    p = W.draw_truth(3000, seed=7)
    obs = orc.synth(p[:1], lam, oracle_lines(c1["lines"], True))[0] + W.draw_noise((4, 128), 1e-3)
    model = orc.synth(p, lam, oracle_lines(c1["lines"], True), threads=NTHREADS)
    w, sig = c1["ga"]["stokes_weight"], c1["ga"]["sigma"]
    want = np.array([orc.chi2(obs, m, w, sig) for m in model])
    _, chi_a = B.me_synth(dev(p), lam, ld, obs_ref=dev(obs), w_over_sigma=w / sig)
    _, chi_b = B.me_synth(dev(p), lam, ld, obs_ref=dev(obs), w_over_sigma=w / sig, want_stokes=False)
    # The two legs are different instantiations since round 2: with the Stokes output the model is formed and subtracted from
    # the reference, without it the residual is the last FMA of the Unno-Rachkovsky tail (as in the fused GA fitness).  Both
    # must meet the fused-fitness tolerance against the oracle, and they differ from each other by
    # binary32 rounding only.
    for chi in (chi_a, chi_b):
        got = chi.cpu().numpy().astype(np.float64)
        assert np.max(np.abs(got - want) / want) < 2e-4
    mutual = float(((chi_a - chi_b).abs() / chi_a).max())
    print("me_synth chi2, with vs without Stokes output: max relative difference %.2e" % mutual)
    assert mutual < 5e-6                                          # measured 2.3e-7
    assert B.me_synth(dev(p[:0]), lam, ld)[0].shape[0] == 0       # empty input


# ---------------------------------------------------------------------------------------------------- GA stages
@pytest.mark.parametrize("pop,k", [(64, 3), (100, 2), (128, 3), (512, 4), (2, 1), (1024, 3)])
def test_ga_init_and_step_bit_exact(B, pop, k):
    G = 20
    cfg = W.ga_config(pop, G, tournament_k=k)
    N, seed, base = 37, 0xABCDEF0123, 4000000000
    g0 = B.ga_init(N, cfg, seed, pixel_id_base=base)
    assert np.array_equal(g0.cpu().numpy(), orc.ga_init(N, pop, seed, pixel_base=base))
    rng = np.random.default_rng(pop)
    genes = rng.random((N, pop, 9)).astype(np.float32)
    chi2 = (rng.random((N, pop)) * 50).astype(np.float32)
    chi2[0, : pop // 2] = chi2[0, 0]                              # ties
    chi2[1, 1] = np.inf
    chi2[2, :] = 7.0
    for t in (1, 7, G):
        got = B.ga_step(dev(genes), dev(chi2), t, cfg, seed, pixel_id_base=base).cpu().numpy()
        want = orc.ga_step(genes, chi2.astype(np.float64), t, cfg, seed, pixel_base=base)
        assert np.array_equal(got, want), (pop, k, t)
    # NaN fitness is treated as +Inf (reading G4)
    chi2n = chi2.copy(); chi2n[3, 0] = np.nan
    chi2i = chi2.copy(); chi2i[3, 0] = np.inf
    assert torch.equal(B.ga_step(dev(genes), dev(chi2n), 2, cfg, seed), B.ga_step(dev(genes), dev(chi2i), 2, cfg, seed))


@pytest.mark.parametrize("which", ["config0", "config1", "full_pattern"])
def test_fused_fitness_vs_oracle(B, which):
    cfgw = W.config0() if which == "config0" else W.config1()
    triplets = which != "full_pattern"
    cfgw = dict(cfgw, triplets=triplets)
    N, pop = 24, cfgw["ga"]["pop"]
    mu = np.linspace(0.1, 1.0, N)
    truth, obs, ln = make_obs(cfgw, N, mu=mu, threads=NTHREADS)
    genes = orc.ga_init(N, pop, seed=11)
    genes[:, 0, :] = 0.0; genes[:, 1, :] = 1.0                      # box corners
    want = orc.ga_fitness(genes, obs, cfgw["lam"], ln, cfgw["ga"], mu=mu, threads=NTHREADS)
    ld = B.line_data_from_workload(cfgw["lines"], triplets)
    got = B.ga_fitness(dev(genes), dev(obs), cfgw["lam"], ld, cfgw["ga"], mu=dev(mu)).cpu().numpy().astype(np.float64)
    rel = np.abs(got - want) / want
    assert rel.max() < 2e-4, rel.max()
    assert np.median(rel) < 1e-5


def test_me_synth_large_damping(B):
    # damping beyond the configs' box: a in (0.5, 0.75] still takes the far-tier polynomials (FAD_FAR_AMAX), a > 0.75 the
    # plain wing series; both must hold the synthesis tolerance, also at the largest eta0
    c1 = W.config1()
    lam = c1["lam"]
    P = 3000
    p = W.draw_truth(P, seed=55, b_lo=1.0, b_hi=3500.0)
    rng = np.random.default_rng(9)
    p[:, 5] = np.concatenate([rng.uniform(0.5, 0.75, P // 3), rng.uniform(0.75, 0.76, P // 3), rng.uniform(0.76, 2.5, P - 2 * (P // 3))])
    p[::2, 3] = 50.0
    ln = oracle_lines(c1["lines"], True)
    ref = orc.synth(p, lam, ln, threads=NTHREADS)
    out, _ = B.me_synth(dev(p), lam, B.line_data_from_workload(c1["lines"], True))
    err = np.abs(out.cpu().numpy() - ref) / (p[:, 7] + p[:, 8])[:, None, None]
    print("forward synthesis: max |dStokes| / I_c = %.2e (north_star bound 2e-5)" % err.max())
    assert err.max() <= 2e-5, (err.max(), p[np.unravel_index(err.argmax(), err.shape)[0]])


def test_me_synth_large_batch_order_is_invisible(B):
    # batches of >= 400 000 vectors are visited in a counting-sort order (tier coherence); every output must sit at its own
    # index and be bit-identical to what the same vector gives in a small (unsorted) batch, with and without chi2
    c1 = W.config1()
    lam = c1["lam"]
    P = 400003
    p = W.draw_truth(P, seed=91, b_lo=1.0, b_hi=3500.0)
    p[:5, 0] = 0.0                                              # B = 0 and extreme keys
    p[5:10, 6] = [-30.0, 30.0, -7.99, 7.99, 0.0]
    mu = np.random.default_rng(4).uniform(0.05, 1.0, P)
    ld = B.line_data_from_workload(c1["lines"], True)
    d_p, d_mu = dev(p), dev(mu)
    obs_ref = dev(orc.synth(p[:1], lam, oracle_lines(c1["lines"], True))[0])
    wos = c1["ga"]["stokes_weight"] / c1["ga"]["sigma"]
    # the ordering scratch is the CALLER's: the library reports its size and allocates nothing itself
    need = B.me_synth_workspace_bytes(P)
    assert need == (2 * P + 32768 + 32) * 4 and B.me_synth_workspace_bytes(399999) == 0 and B.me_synth_workspace_bytes(2 ** 31) == 0
    big, chi_big = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos,
                              workspace=torch.empty((need,), dtype=torch.uint8, device="cuda"))
    plain, chi_plain = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos, workspace=False)   # me_synth proper
    assert torch.equal(big, plain) and torch.equal(chi_big, chi_plain)
    short, chi_short = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos,
                                  workspace=torch.empty((need - 16,), dtype=torch.uint8, device="cuda"))   # too small: ignored
    assert torch.equal(big, short) and torch.equal(chi_big, chi_short)
    del plain, short
    # the chi2-only instantiation (no [P,4,L] output, no transpose tile, 5 CTAs per SM), ordered and in index order: the fused
    # residual of its tail rounds like the explicit subtraction of the output instantiation or differs by an ulp of chi2
    for ws in (None, False):
        _, chi_only = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos, want_stokes=False, workspace=ws)
        assert torch.allclose(chi_only, chi_big, rtol=2e-4, atol=0.0)
        if ws is None:
            chi_only_ordered = chi_only
    assert torch.equal(chi_only, chi_only_ordered)
    for s in (0, 150000, 300000):
        e = min(s + 150000, P)
        small, chi_small = B.me_synth(d_p[s:e].contiguous(), lam, ld, mu=d_mu[s:e].contiguous(), obs_ref=obs_ref, w_over_sigma=wos)
        assert torch.equal(big[s:e], small) and torch.equal(chi_big[s:e], chi_small)
    # and a sample against the oracle
    idx = np.arange(0, P, 4000)
    ref = orc.synth(p[idx], lam, oracle_lines(c1["lines"], True), mu=mu[idx], threads=NTHREADS)
    err = np.abs(big.cpu().numpy()[idx] - ref) / (p[idx, 7] + mu[idx] * p[idx, 8])[:, None, None]
    print("forward synthesis: max |dStokes| / I_c = %.2e (north_star bound 2e-5)" % err.max())
    assert err.max() <= 2e-5
