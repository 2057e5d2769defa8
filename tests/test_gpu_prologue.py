"""GPU parity of the per-pixel prologue (ga_cfg.prologue; readings W1, P1 of DESIGN.md): inverse-max weights
(eq. 20-23) and the polarity restriction of the inclination."""
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


@pytest.mark.parametrize("flags", [0, 1, 2, 3])
@pytest.mark.parametrize("which", ["config0", "config1"])
def test_prologue_hook_vs_oracle(B, which, flags):
    c = W.config0() if which == "config0" else W.config1()
    N = 300
    truth, obs, ln = make_obs(c, N, threads=NTHREADS)
    obs[5, 2] = 0.0                                            # an empty Stokes parameter: floored at sigma
    obs[6, 3] = 0.0                                            # no V signal at all: argmax = argmin = 0 -> [90, 180]
    cfg = dict(c["ga"], prologue=flags)
    want = orc.prologue(obs, cfg)
    ld = B.line_data_from_workload(c["lines"], True)
    got = B.ga_prologue(dev(obs), c["lam"], ld, cfg).cpu().numpy().astype(np.float64)
    assert np.array_equal(got[:, 4:6], want[:, 4:])           # the polarity box is an exact decision
    assert np.all(got[:, 6:] == 0.0)                          # no seeds asked for
    assert np.max(np.abs(got[:, :4] - want[:, :4]) / want[:, :4]) < 1e-6
    if flags & 2:
        strong = truth[:, 0] > 800.0                           # strong fields: the lobe order gives the true polarity
        assert np.mean((want[strong, 5] <= 90.0) == (truth[strong, 1] < 90.0)) > 0.97


@pytest.mark.parametrize("which,variant", [("config0", 0), ("config1", 0), ("config1", 1)])
def test_seeds_hook_vs_oracle(B, which, variant):
    c = W.config0() if which == "config0" else W.config1()
    N = 400
    truth, obs, ln = make_obs(c, N, threads=NTHREADS)
    cfg = dict(c["ga"], prologue=4, variant=variant)
    want = orc.seeds(obs, c["lam"], ln, cfg)
    ld = B.line_data_from_workload(c["lines"], True)
    got = B.ga_prologue(dev(obs), c["lam"], ld, cfg).cpu().numpy().astype(np.float64)
    big = np.abs(want[:, 0]) > 5.0
    assert np.max(np.abs(got[big, 6] - want[big, 0]) / np.abs(want[big, 0])) < 2e-3     # B_los: FP32 centroid differences
    assert np.max(np.abs(got[:, 6] - want[:, 0])) < 0.05                                 # ... a few hundredths of a Gauss
    gene = (lambda q: 64.0 * q) if variant else (lambda q: (q.astype(np.float32) / np.float32(1023.0)).astype(np.float64))
    same_b = got[:, 7] == gene(want[:, 1])
    same_g = got[:, 8] == gene(want[:, 2])
    assert same_b.mean() > 0.97 and same_g.mean() > 0.97      # 10-bit quantisation: equal except at a rounding boundary / B_los ~ 0
    off = np.abs(got[~same_b, 7] - gene(want[~same_b, 1]))
    assert off.size == 0 or off.max() <= (64.0 if variant else 1.01 / 1023.0)           # and then by one step only


def test_inversion_with_seeds_parity(B):
    c0 = W.config0()
    # 256 pixels, not 64: the identical-optimum fraction of the binary-coded variant is ~0.90, and on 64 pixels its sampling
    # error (+-4.5 %) straddles the 0.85 floor.  Bisected in round 2 on these 256 pixels (and on their first 64, the former
    # sample): kernel of 14cb8fd, the last that met 0.85: 0.906 (0.859); round-1 final kernel: 0.902 (0.828); round-2 kernel:
    # 0.902 (0.828).  Round 1 answered the 55 -> 53 of 64 by lowering the floor to 0.75; the agreement itself had not moved.
    N = 256
    truth, obs, ln = make_obs(c0, N, threads=NTHREADS)
    ld = B.line_data_from_workload(c0["lines"], True)
    for variant in (0, 1):
        ga = dict(c0["ga"], prologue=7, variant=variant)
        res = orc.ga_invert(obs, c0["lam"], ln, ga, seed=W.SEED_GA, threads=NTHREADS)
        gp, gc = B.ga_invert(dev(obs), c0["lam"], ld, ga, W.SEED_GA)
        gc = gc.cpu().numpy().astype(np.float64)
        same = np.abs(gc - res["chi2"]) <= 2e-4 * res["chi2"]
        # reading G4: trajectories part only where an FP32 and an FP64 chi2 compare differently.  The identical-optimum floor
        # is 0.85, as it was before round 1's far-tier commit lowered it to 0.75; measured on this sample 0.996
        # (real-coded) and 0.902 (binary-coded), sampling error +-2.2 %.  north_star's statistical criterion (median chi2
        # within 1 %) is asserted beside it.
        print("seeded inversion, variant %d: identical-optimum fraction %.3f" % (variant, same.mean()))
        assert same.mean() >= 0.85, (variant, same.mean())
        assert abs(np.median(gc) - np.median(res["chi2"])) <= 0.01 * np.median(res["chi2"])
    # zero generations, everything but (B, gamma) fixed at the truth: the centre-of-gravity member wins on both sides
    strong = np.flatnonzero((truth[:, 0] > 800.0) & (np.abs(np.cos(np.radians(truth[:, 1]))) > 0.8))[:6]
    for n in strong:
        ga = W.ga_config(32, 0, prologue=4)
        for j in range(2, 9):
            ga["lo"][j] = ga["hi"][j] = truth[n, j]
        r = orc.ga_invert(obs[n:n + 1], c0["lam"], ln, ga, seed=2, pixel_base=int(n))
        p, c = B.ga_invert(dev(obs[n:n + 1]), c0["lam"], ld, ga, 2, pixel_id_base=int(n))
        assert abs(float(c[0]) - r["chi2"][0]) <= 2e-4 * r["chi2"][0]
        assert np.allclose(p.cpu().numpy()[0], r["params"][0], rtol=2e-3, atol=1e-3)


def test_inversion_with_prologue_parity(B):
    c0 = W.config0()
    N = 64
    truth, obs, ln = make_obs(c0, N, threads=NTHREADS)
    ga = dict(c0["ga"], prologue=3)
    res = orc.ga_invert(obs, c0["lam"], ln, ga, seed=W.SEED_GA, threads=NTHREADS)
    ld = B.line_data_from_workload(c0["lines"], True)
    gp_d, gc_d = B.ga_invert(dev(obs), c0["lam"], ld, ga, W.SEED_GA)
    gp, gc = gp_d.cpu().numpy().astype(np.float64), gc_d.cpu().numpy().astype(np.float64)
    same = np.abs(gc - res["chi2"]) <= 2e-4 * res["chi2"]
    assert same.mean() >= 0.9, same.mean()
    assert abs(np.median(gc) - np.median(res["chi2"])) <= 0.01 * np.median(res["chi2"])
    pro = orc.prologue(obs, ga)
    assert np.all(gp[:, 1] >= pro[:, 4] - 1e-4) and np.all(gp[:, 1] <= pro[:, 5] + 1e-4)     # inside the polarity box
    # chi2 returned = eq. 16 of the returned parameters with the per-pixel weights: the oracle's optimum re-evaluated by the
    # oracle with the prologue weights equals its own chi2 (pins the weights inside the oracle's GA) ...
    model = orc.synth(res["params"], c0["lam"], ln, threads=NTHREADS)
    chk = np.array([orc.chi2(o, m, w[:4], ga["sigma"]) for o, m, w in zip(obs, model, pro)])
    assert np.allclose(chk, res["chi2"], rtol=1e-12)
    # ... and the GPU's chi2 is reproduced by the library's own per-pixel evaluator (same weights, same box)
    _, chk_g = B.ga_uncertainty(dev(obs), gp_d, c0["lam"], ld, ga)
    assert float(((gc_d - chk_g).abs() / chk_g).max()) < 1e-5
    # flags off: bit-identical to a run that never heard of the prologue
    a = B.ga_invert(dev(obs), c0["lam"], ld, c0["ga"], W.SEED_GA)
    b = B.ga_invert(dev(obs), c0["lam"], ld, dict(c0["ga"], prologue=0), W.SEED_GA)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    # the polarity restriction halves the inclination domain: it must not hurt strong-field recovery
    strong = truth[:, 0] > 800.0
    assert np.median(np.abs(gp[strong, 1] - truth[strong, 1])) < 5.0


@pytest.mark.parametrize("which,flags,variant", [("config0", 8, 0), ("config1", 8, 0), ("config1", 2 | 8, 0), ("config1", 2 | 8, 1)])
def test_auer_member_hook_vs_oracle(B, which, flags, variant):
    # reading S2: the stored genes (B, gamma, chi) of the weak-field member, FP32 on the device against
    # the FP64 oracle from the same binary32 observations; with bit 2 the inclination box is the polarity-cut one (reading P1)
    c = W.config0() if which == "config0" else W.config1()
    N = 400
    truth, obs, ln = make_obs(c, N, threads=NTHREADS)
    cfg = dict(c["ga"], prologue=flags, variant=variant)
    box = orc.prologue(obs, cfg)
    want = orc.seed_auer(obs, c["lam"], ln, cfg, glo=box[:, 4], ghi=box[:, 5])
    ld = B.line_data_from_workload(c["lines"], True)
    got = B.ga_prologue(dev(obs), c["lam"], ld, cfg).cpu().numpy().astype(np.float64)
    assert np.all(got[:, 6:9] == 0.0)                                   # bit 4 clear: no centre-of-gravity member
    gene = (lambda q: 64.0 * q) if variant else (lambda q: (q.astype(np.float32) / np.float32(1023.0)).astype(np.float64))
    step = 64.0 if variant else 1.01 / 1023.0
    frac = []
    for k, name in enumerate(("B", "gamma", "chi")):
        same = got[:, 9 + k] == gene(want[:, 4 + k])
        off = np.abs(got[~same, 9 + k] - gene(want[~same, 4 + k]))
        if name == "chi":                                               # 0 and 180 deg are the same azimuth: the two ends of the box
            off = np.minimum(off, np.abs(off - (65472.0 if variant else 1.0)))
        frac.append(same.mean())
        # 10-bit quantisation: equal except at a rounding boundary, and then by one step
        assert off.size == 0 or np.mean(off <= step) > 0.9, (name, np.sort(off)[-5:])
    print("Auer genes equal to the oracle's (B, gamma, chi): %.3f %.3f %.3f" % tuple(frac))
    assert min(frac) > 0.95, frac
    if flags & 2:                                                       # consistent with the polarity box
        lo, hi = box[:, 4], box[:, 5]
        gam = lo + (hi - lo) * (got[:, 10] / 65535.0 if variant else got[:, 10])
        assert np.all(gam >= lo - 1e-4) and np.all(gam <= hi + 1e-4)


def test_inversion_with_all_prologue_members_parity(B):
    # every flag of the paper's prologue at once (weights, polarity, centre-of-gravity + non-magnetic + Auer members);
    # 256 pixels for the same reason as in test_inversion_with_seeds_parity
    c0 = W.config0()
    N = 256
    truth, obs, ln = make_obs(c0, N, threads=NTHREADS)
    ld = B.line_data_from_workload(c0["lines"], True)
    for variant in (0, 1):
        ga = dict(c0["ga"], prologue=15, variant=variant)
        res = orc.ga_invert(obs, c0["lam"], ln, ga, seed=W.SEED_GA, threads=NTHREADS)
        gp, gc = B.ga_invert(dev(obs), c0["lam"], ld, ga, W.SEED_GA)
        gc = gc.cpu().numpy().astype(np.float64)
        same = np.abs(gc - res["chi2"]) <= 2e-4 * res["chi2"]
        print("all prologue members, variant %d: identical-optimum fraction %.3f" % (variant, same.mean()))
        assert same.mean() >= 0.85, (variant, same.mean())
        assert abs(np.median(gc) - np.median(res["chi2"])) <= 0.01 * np.median(res["chi2"])
    # zero generations, thermodynamics fixed at the truth: the Auer member wins on both sides, same parameters
    weak = np.flatnonzero((truth[:, 0] > 150.0) & (truth[:, 0] < 900.0))[:6]
    for n in weak:
        ga = W.ga_config(32, 0, prologue=8)
        for j in range(3, 9):
            ga["lo"][j] = ga["hi"][j] = truth[n, j]
        r = orc.ga_invert(obs[n:n + 1], c0["lam"], ln, ga, seed=2, pixel_base=int(n))
        p, c = B.ga_invert(dev(obs[n:n + 1]), c0["lam"], ld, ga, 2, pixel_id_base=int(n))
        assert abs(float(c[0]) - r["chi2"][0]) <= 2e-4 * r["chi2"][0]
        assert np.allclose(p.cpu().numpy()[0], r["params"][0], rtol=2e-3, atol=1e-3)
    # too small a population for the member is refused, nothing launched
    with pytest.raises(B.MeError):
        B.ga_invert(dev(obs[:1]), c0["lam"], ld, W.ga_config(3, 1, prologue=8), 1)
