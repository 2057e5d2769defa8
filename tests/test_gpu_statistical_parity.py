"""north_star's statistical parity of the whole inversion, at sample sizes where the medians mean something.

The CUDA path (ga_invert through the C ABI) and the CPU oracle invert the SAME seeded pixels (oracle-synthesised
observations + seeded noise, rounded to binary32) with the SAME Philox streams (global pixel ids), and north_star's
criteria are asserted as written: median chi2 within 1 %, median |dB|, |dgamma|, |dchi| (mod 180 deg), |dv| against the
generating truth each within 5 % of the oracle's.  Additionally the fraction of pixels that end on the identical optimum
is reported (the only place the trajectories can part is the `<` on binary32 vs binary64 chi2, reading G4).

Sample sizes: config 1 on 1024 pixels, config 3 (the north_star target: full-disc ids, mask, mu, 80 % quiet / 20 % active,
200 generations) on 640 pixels; ME_PARITY_PIXELS=<n> scales both (SURVEY.md 8(d) asks for 4096 where possible:
`ME_PARITY_PIXELS=4096 python -m pytest tests/test_gpu_statistical_parity.py -m gpu -s`).  Each run writes its table to
gpurun_out/parity_<config>.md when that folder exists.  Nothing computed by the CUDA path is an oracle input.
"""
import os
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from helpers import oracle_lines
from oracle import api as orc
from paper_1208_0302_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
NTHREADS = max(1, (os.cpu_count() or 1))
SCALE = int(os.environ.get("ME_PARITY_PIXELS", "0"))
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1208_0302_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def dev(a, dtype=np.float32):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def errors(p, truth):
    dchi = np.abs(p[:, 2] - truth[:, 2]) % 180.0
    return {"B [G]": np.abs(p[:, 0] - truth[:, 0]), "gamma [deg]": np.abs(p[:, 1] - truth[:, 1]),
            "chi [deg]": np.minimum(dchi, 180.0 - dchi), "v_los [km/s]": np.abs(p[:, 6] - truth[:, 6])}


def invert_both(B, cfg, ids, truth, mu, noise_stream):
    """Both sides invert pixel k under global id ids[k]; one call per run of consecutive ids."""
    n = ids.size
    ln = oracle_lines(cfg["lines"], True)
    clean = orc.synth(truth, cfg["lam"], ln, mu=mu, threads=NTHREADS)
    obs = (clean + W.draw_noise(clean.shape, cfg["sigma"], stream=noise_stream)).astype(np.float32)
    ld = B.line_data_from_workload(cfg["lines"], True)
    d_obs, d_mu = dev(obs), dev(mu)
    runs = np.split(np.arange(n), np.flatnonzero(np.diff(ids) != 1) + 1)
    gp, gc = np.empty((n, 9)), np.empty(n)
    t0 = time.perf_counter()
    for r in runs:
        p, c = B.ga_invert(d_obs[r[0]:r[-1] + 1].contiguous(), cfg["lam"], ld, cfg["ga"], W.SEED_GA,
                           mu=d_mu[r[0]:r[-1] + 1].contiguous(), pixel_id_base=int(ids[r[0]]))
        gp[r], gc[r] = p.cpu().numpy(), c.cpu().numpy()
    torch.cuda.synchronize()
    t_gpu = time.perf_counter() - t0
    obs64 = obs.astype(np.float64)
    op, oc = np.empty((n, 9)), np.empty(n)
    single = len(runs) == 1

    def one(r):
        return r, orc.ga_invert(obs64[r[0]:r[-1] + 1], cfg["lam"], ln, cfg["ga"], seed=W.SEED_GA, mu=mu[r[0]:r[-1] + 1],
                                pixel_base=int(ids[r[0]]), threads=NTHREADS if single else 1)
    t0 = time.perf_counter()
    with ThreadPoolExecutor(1 if single else NTHREADS) as ex:        # ctypes releases the GIL
        for r, res in ex.map(one, runs):
            op[r], oc[r] = res["params"], res["chi2"]
    return gp, gc, op, oc, t_gpu, time.perf_counter() - t0, len(runs)


def judge(name, label, truth, gp, gc, op, oc, t_gpu, t_orc, ncalls, min_same):
    """north_star's criteria, asserted as written; the table goes to gpurun_out/parity_<name>.md when that folder exists."""
    n = gc.size
    same = (np.abs(gc - oc) <= 2e-4 * oc) & np.all(np.abs(gp - op) <= 1e-4 * (np.abs(op) + 1.0), axis=1)
    mg, mo = np.median(gc), np.median(oc)
    rows = ["# Statistical parity - %s\n" % label,
            "Command: `ME_PARITY_PIXELS=%d python -m pytest tests/test_gpu_statistical_parity.py -m gpu -s -k %s` "
            "(one B200; oracle on %d host threads)\n" % (SCALE, name, NTHREADS),
            "%d pixels; CUDA path %.2f s (%d ga_invert calls), oracle %.0f s.\n" % (n, t_gpu, ncalls, t_orc),
            "| quantity | CUDA path | oracle | relative difference | north_star bound |", "|---|---|---|---|---|",
            "| median chi2 | %.5f | %.5f | %.3f %% | 1 %% |" % (mg, mo, 100 * abs(mg - mo) / mo)]
    eg, eo = errors(gp, truth), errors(op, truth)
    rel = {}
    for k in eg:
        x, y = np.median(eg[k]), np.median(eo[k])
        rel[k] = abs(x - y) / y
        rows.append("| median abs. error of %s vs truth | %.5g | %.5g | %.3f %% | 5 %% |" % (k, x, y, 100 * rel[k]))
    rows.append("| pixels ending on the identical optimum | %.2f %% | | | |" % (100 * same.mean()))
    worst = np.max(np.abs(gc - oc)[~same] / oc[~same]) if (~same).any() else 0.0
    rows.append("| max relative chi2 difference among the others | %.3g | | | |" % worst)
    text = "\n".join(rows) + "\n"
    print("\n" + text)
    out_dir = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out_dir):
        with open(os.path.join(out_dir, "parity_%s.md" % name), "w") as fh:
            fh.write(text)
    assert np.all(np.isfinite(gc)) and np.all(np.isfinite(gp))
    assert abs(mg - mo) <= 0.01 * mo, (mg, mo)                       # north_star: median chi2 within 1 %
    for k, r in rel.items():
        assert r <= 0.05, (k, r)                                     # north_star: each median error within 5 % of the oracle's
    assert same.mean() >= min_same, same.mean()


def test_config1_statistical_parity(B):
    """BASELINE config 1 (iid prior draws, two triplets, L = 128, pop 128, 100 generations)."""
    n = SCALE or 1024
    cfg = W.config1()
    truth = W.draw_truth(n, seed=W.SEED_TRUTH, stream=11)
    ids, mu = np.arange(n), np.ones(n)
    out = invert_both(B, cfg, ids, truth, mu, noise_stream=11)
    # The identical-optimum fraction is a diagnostic, not a north_star criterion: it measures how often the one binary32-vs-
    # binary64 `<` (reading G4) parts two chaotic trajectories.  Measured on these 1024 pixels with the round-1 kernel:
    # 90.3 % (sampling noise +- 0.9 %; 93.9 % with the more accurate r1f Voigt tiers).  Floor 0.85, fixed before any
    # round-2 kernel change; a kernel that falls below it has lost accuracy and must say so, not move the floor.
    judge("config1", "config1: %d iid prior draws, two triplets, L = 128, pop 128, 100 generations" % n, truth, *out, min_same=0.85)


def test_config3_statistical_parity(B):
    """BASELINE config 3, the north_star target: pixels of the 2048^2 full-disc map at their global ids, mu per pixel,
    80 % quiet Sun (B log-U[1,200] G) / 20 % active region (B 500-3500 G), B box [1,3500] G, 200 generations."""
    n = (SCALE // 2) or 640
    cfg = W.config3()
    mask, mu_all, truth_all, active = W.fulldisc_truth(cfg["n_side"], cfg["radius"])
    on = mask.astype(bool)
    q, ac = np.flatnonzero(on & ~active), np.flatnonzero(on & active)
    nq = int(0.8 * n)
    ids = np.concatenate([q[:: max(1, q.size // nq)][:nq], ac[:: max(1, ac.size // (n - nq))][: n - nq]])
    truth, mu = truth_all[ids], mu_all[ids]
    out = invert_both(B, cfg, ids, truth, mu, noise_stream=11)
    # 200 generations on mostly weak-field pixels, whose chi2 surface is flat in the angles, give the single
    # binary32-vs-binary64 `<` (reading G4) more occasions to part the trajectories than config 1 does: the identical-
    # optimum fraction is reported, and only a floor is asserted; north_star's population statistics are the criterion.
    judge("config3", "config3: 2048^2 full-disc map, %d quiet + %d active-region on-disc pixels at their global ids, mu per "
          "pixel, 200 generations" % (min(nq, ids.size), ids.size - min(nq, ids.size)), truth, *out, min_same=0.5)
