"""The product calls under CUDA graph capture ("no allocation visible to the caller", no synchronisation).

include/me.h states that ga_invert, me_synth and me_synth_static allocate nothing and do not synchronise.  A stream capture is
the strictest check of that statement the runtime offers: cudaMalloc, cudaFree, a device or stream synchronisation or a launch
on another stream invalidates the capture and the call returns an error.  The replayed graph must reproduce the eager result
bit for bit (same kernels, same descriptors by value).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1208_0302_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1208_0302_b200 import binding, build
    build.build()
    return binding


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).cuda()


def _observations(B, cfg, n, seed):
    """Noisy observations made by the CUDA path itself (this file compares the CUDA path with itself; parity is elsewhere)."""
    ld = B.line_data_from_workload(cfg["lines"], True)
    truth = W.draw_truth(n, seed=seed)
    clean, _ = B.me_synth(dev(truth), cfg["lam"], ld)
    noise = W.draw_noise(tuple(clean.shape), 1e-3)
    return ld, (clean + dev(noise)).contiguous()


def test_ga_invert_is_capturable_and_replays_bit_identically(B):
    c0 = W.config0()
    ld, obs = _observations(B, c0, 64, 11)
    n, m = obs.shape[0], ld.n_params
    eager_p, eager_c = B.ga_invert(obs, c0["lam"], ld, c0["ga"], W.SEED_GA)
    torch.cuda.synchronize()
    out_p = torch.zeros((n, m), dtype=torch.float32, device="cuda")
    out_c = torch.zeros((n,), dtype=torch.float32, device="cuda")
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):                                   # capture: nothing runs yet
        B.ga_invert(obs, c0["lam"], ld, c0["ga"], W.SEED_GA, out_params=out_p, out_chi2=out_c)
    assert float(out_c.abs().sum()) == 0.0
    for _ in range(2):
        out_p.zero_(); out_c.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out_p, eager_p) and torch.equal(out_c, eager_c)
    # new observations in the SAME buffer: the graph reads the buffer, not a copy
    _, obs2 = _observations(B, c0, 64, 12)
    eager2_p, eager2_c = B.ga_invert(obs2, c0["lam"], ld, c0["ga"], W.SEED_GA)
    obs.copy_(obs2)
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out_p, eager2_p) and torch.equal(out_c, eager2_c) and not torch.equal(eager2_c, eager_c)


def test_me_synth_static_is_capturable(B):
    c1 = W.config1()
    lam, L = c1["lam"], len(c1["lam"])
    ld = B.line_data_from_workload(c1["lines"], True)
    wos = c1["ga"]["stokes_weight"] / c1["ga"]["sigma"]
    P = 400003                                                  # large enough for the ordered visit through the fixed scratch array
    p = W.draw_truth(P, seed=21, b_lo=1.0, b_hi=3500.0)
    d_p = dev(p)
    obs_ref = B.me_synth(d_p[:1].contiguous(), lam, ld)[0][0].contiguous()
    chi = torch.zeros((P,), dtype=torch.float32, device="cuda")
    # once eagerly: the scratch array's address is looked up once per device (cudaGetSymbolAddress), outside any capture
    B.me_synth_static(d_p, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi)
    torch.cuda.synchronize()
    eager = chi.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        B.me_synth_static(d_p, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi)
    for _ in range(2):
        chi.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(chi, eager)
