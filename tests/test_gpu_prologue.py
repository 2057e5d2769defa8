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
    got = B.ga_prologue(dev(obs), cfg).cpu().numpy().astype(np.float64)
    assert np.array_equal(got[:, 4:], want[:, 4:])            # the polarity box is an exact decision
    assert np.max(np.abs(got[:, :4] - want[:, :4]) / want[:, :4]) < 1e-6
    if flags & 2:
        strong = truth[:, 0] > 800.0                           # strong fields: the lobe order gives the true polarity
        assert np.mean((want[strong, 5] <= 90.0) == (truth[strong, 1] < 90.0)) > 0.97


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
