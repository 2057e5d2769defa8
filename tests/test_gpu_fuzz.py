"""Randomised sweep over the template specialisations of the library (lines 1..4, effective triplets / full Zeeman patterns,
9 / 11 parameters, odd and even L, population sizes around the block-size thresholds): for each drawn configuration the
fused fitness (ga_fitness hook), me_synth and a short inversion are compared with the oracle.  Seeded, so every run
checks the same 14 configurations."""
import os

import numpy as np
import pytest

from helpers import oracle_lines
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


def _draw(k):
    rng = np.random.default_rng(1000 + k)
    n_lines = int(rng.integers(1, 5))
    base = [W.FE_6301, W.FE_6302]
    lines = []
    for i in range(n_lines):
        l = dict(base[i % 2])
        l["lambda0"] = l["lambda0"] + 0.35 * (i // 2)               # a shifted copy of the multiplet for lines 3, 4
        l["strength"] = float(rng.uniform(0.3, 3.6))
        lines.append(l)
    triplets = bool(rng.integers(0, 2))
    npar = int(rng.choice([9, 11]))
    L = int(rng.choice([7, 31, 50, 64, 97, 128, 200]))
    step = float(rng.uniform(0.015, 0.04))
    centre = float(np.mean([l["lambda0"] for l in lines]))
    pop = int(rng.choice([2, 33, 64, 65, 128, 129, 300]))
    return lines, triplets, npar, W.grid(centre, L, step), pop, rng


@pytest.mark.parametrize("k", range(14))
def test_random_configuration(B, k):
    lines, triplets, npar, lam, pop, rng = _draw(k)
    ln = oracle_lines(lines, triplets)
    nm = nm_d = None
    if npar == 11:
        nm32 = orc.synth(W.NM_PARAMS[None, :], lam, ln)[0, 0].astype(np.float32)
        nm, nm_d = nm32.astype(np.float64), dev(nm32)
    ld = B.line_data_from_workload(lines, triplets, n_params=npar, nm_profile=nm_d)
    N = 3
    mu = rng.uniform(0.1, 1.0, N)
    sigma = float(rng.choice([1e-3, 3e-3]))
    ga = W.ga_config(pop, 3, sigma=sigma, b_lo=1.0, b_hi=3500.0, npar=npar, tournament_k=int(rng.integers(1, 5)),
                     variant=int(rng.integers(0, 2)), prologue=0)
    truth = W.draw_truth(N, seed=50 + k, b_lo=1.0, b_hi=3500.0, npar=npar)
    clean = orc.synth(truth, lam, ln, mu=mu, nm_profile=nm, threads=NTHREADS)
    # forward synthesis
    out, _ = B.me_synth(dev(truth), lam, ld, mu=dev(mu))
    cont = (truth[:, 7] + mu * truth[:, 8])[:, None, None]
    assert np.max(np.abs(out.cpu().numpy() - clean) / cont) <= 2e-5
    # fused fitness of a generation-0 population (codes or genes, per the variant)
    obs = (clean + W.draw_noise(clean.shape, sigma, stream=k)).astype(np.float32).astype(np.float64)
    genes = orc.ga_init(N, pop, seed=k, npar=npar, variant=ga["variant"])
    want = orc.ga_fitness(genes, obs, lam, ln, ga, mu=mu, threads=NTHREADS, nm_profile=nm)
    got = B.ga_fitness(dev(genes), dev(obs), lam, ld, ga, mu=dev(mu)).cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got - want) / want) < 2e-4
    # three generations of the whole inversion, with the prologue on for odd k
    ga2 = dict(ga, prologue=3 if k % 2 else 0)
    res = orc.ga_invert(obs, lam, ln, ga2, seed=9 + k, mu=mu, threads=NTHREADS, nm_profile=nm, pixel_base=77)
    gp, gc = B.ga_invert(dev(obs), lam, ld, ga2, 9 + k, mu=dev(mu), pixel_id_base=77)
    gc = gc.cpu().numpy().astype(np.float64)
    # three generations leave little room for the trajectories to part: the optimum is the same individual
    assert np.max(np.abs(gc - res["chi2"]) / res["chi2"]) < 2e-4, (gc, res["chi2"])
    assert np.allclose(gp.cpu().numpy(), res["params"], rtol=2e-4, atol=2e-4)
