"""me_synth_static: the entry point that allocates nothing (include/me.h), against the existing me_synth / me_synth_ws paths.

Collected LAST on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, and a failure
here must not hide the parity tests.  Passes alone in a fresh process and after the other tests: it depends on no state but the
library's own fixed scratch array, whose stale contents are part of what is tested (two calls in a row, the second on another
batch of another size).
"""
import ctypes as C

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


def _batch(P, seed):
    p = W.draw_truth(P, seed=seed, b_lo=1.0, b_hi=3500.0)
    mu = np.random.default_rng(seed).uniform(0.05, 1.0, P)
    return dev(p), dev(mu)


def test_static_scratch_entry_point_matches_existing_paths_twice(B):
    c1 = W.config1()
    lam, L = c1["lam"], len(c1["lam"])
    ld = B.line_data_from_workload(c1["lines"], True)
    wos = c1["ga"]["stokes_weight"] / c1["ga"]["sigma"]
    assert B.me_synth_static_max_vectors() == 2 ** 21
    # an observed profile for the chi2 leg, made by the CUDA path itself (this test compares CUDA paths with each other; parity
    # with the oracle is tests/test_gpu_parity.py's business)
    p0, mu0 = _batch(1, 5)
    obs_ref = B.me_synth(p0, lam, ld, mu=mu0)[0][0].contiguous()
    # two calls in a row through the fixed array: both >= 400 000 vectors, so both use the scratch (counting-sort order and task
    # counter); the second batch is another draw of another size, so that keys, permutation, histogram and counter left by
    # the first call are all stale
    for P, seed in ((400003, 91), (524289, 92)):
        d_p, d_mu = _batch(P, seed)
        out = torch.empty((P, 4, L), dtype=torch.float32, device="cuda")
        chi = torch.empty((P,), dtype=torch.float32, device="cuda")
        mem = torch.cuda.memory_allocated()
        B.me_synth_static(d_p, lam, ld, mu=d_mu, out_stokes=out, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == mem                      # nothing came from torch's allocator either
        # the existing paths: me_synth_ws with a caller workspace (same ordered visit), and me_synth proper (index order).
        # Tolerance: the one tests/test_gpu_parity.py::test_me_synth_large_batch_order_is_invisible uses between these
        # paths, bit-identity (every vector is computed on its own, whatever the visiting order)
        ws, chi_ws = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos)
        assert torch.equal(out, ws) and torch.equal(chi, chi_ws)
        del ws, chi_ws
        plain, chi_plain = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos, workspace=False)
        assert torch.equal(out, plain) and torch.equal(chi, chi_plain)
        assert torch.isfinite(out).all() and torch.isfinite(chi).all()
        del plain, chi_plain, out, chi
    # a small batch needs no scratch and takes the same entry point; chi2-only form
    P = 1000
    d_p, d_mu = _batch(P, 93)
    chi = torch.empty((P,), dtype=torch.float32, device="cuda")
    B.me_synth_static(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi)
    _, chi_plain = B.me_synth(d_p, lam, ld, mu=d_mu, obs_ref=obs_ref, w_over_sigma=wos, want_stokes=False, workspace=False)
    assert torch.equal(chi, chi_plain)


def test_static_scratch_entry_point_at_its_maximum_size(B):
    # exactly me_synth_static_max_vectors() vectors: the batch whose workspace fills the fixed array to its last int (chi2-only
    # form: a [P,4,L] output of that batch would be 4.3 GB); and P = 0 is a no-op that touches nothing
    c1 = W.config1()
    lam = c1["lam"]
    ld = B.line_data_from_workload(c1["lines"], True)
    wos = c1["ga"]["stokes_weight"] / c1["ga"]["sigma"]
    p0, mu0 = _batch(1, 5)
    obs_ref = B.me_synth(p0, lam, ld, mu=mu0)[0][0].contiguous()
    P = B.me_synth_static_max_vectors()
    assert B.me_synth_workspace_bytes(P) == (2 * P + 32768 + 32) * 4          # = the array's size (include/me.h: 16.1 MiB)
    rng = np.random.default_rng(94)
    base = W.draw_truth(4096, seed=94, b_lo=1.0, b_hi=3500.0)
    d_p = dev(base[rng.integers(0, 4096, P)])                                  # 2 097 152 vectors drawn from 4096 distinct ones
    chi = torch.full((P,), float("nan"), dtype=torch.float32, device="cuda")
    B.me_synth_static(d_p, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=chi)
    _, chi_ws = B.me_synth(d_p, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, want_stokes=False)
    assert torch.equal(chi, chi_ws) and torch.isfinite(chi).all()
    empty = torch.empty((0, 9), dtype=torch.float32, device="cuda")
    B.me_synth_static(empty, lam, ld, obs_ref=obs_ref, w_over_sigma=wos, out_chi2=torch.empty((0,), dtype=torch.float32, device="cuda"))


def test_static_scratch_entry_point_refuses_batches_beyond_its_array(B):
    lib = B.lib()
    pmax = B.me_synth_static_max_vectors()
    c1 = W.config1()
    ld = B.line_data_from_workload(c1["lines"], True)
    lam = np.ascontiguousarray(c1["lam"], dtype=np.float64)
    small = torch.zeros((16,), dtype=torch.float32, device="cuda")         # never read: the size check comes first
    rc = lib.me_synth_static(C.c_void_p(small.data_ptr()), C.c_int64(pmax + 1), None, lam.ctypes.data_as(C.POINTER(C.c_double)),
                             C.c_int(lam.size), C.byref(ld.c), C.c_void_p(small.data_ptr()), None, None, None, None)
    assert rc == -6 and b"me_synth_static_max_vectors" in lib.me_strerror(rc)
    with pytest.raises(B.MeError):
        B._check(rc, "me_synth_static")
