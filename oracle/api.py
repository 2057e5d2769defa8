"""oracle/api.py — TEST INFRASTRUCTURE. ctypes front end of the CPU oracle (oracle/liboracle.so).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Everything is numpy float64 in, float64 out; genes are float32 (reading G1).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None
NPAR = 9


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_lande_g.restype = C.c_double
        _lib.orc_g_eff.restype = C.c_double
        _lib.orc_chi2.restype = C.c_double
        _lib.orc_lande_g.argtypes = [C.c_double] * 3
        _lib.orc_g_eff.argtypes = [C.c_double] * 4
    return _lib


def hardware_threads():
    return int(lib().orc_hardware_threads())


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def faddeeva(z):
    z = np.asarray(z, dtype=np.complex128)
    re, im = _f64(z.real.ravel()), _f64(z.imag.ravel())
    wr, wi = np.empty_like(re), np.empty_like(im)
    lib().orc_faddeeva(_p(re, C.c_double), _p(im, C.c_double), C.c_int64(re.size), _p(wr, C.c_double), _p(wi, C.c_double))
    return (wr + 1j * wi).reshape(z.shape)


def lande_g(S, L, J):
    return lib().orc_lande_g(S, L, J)


def g_eff(gl, Jl, gu, Ju):
    return lib().orc_g_eff(gl, Jl, gu, Ju)


def zeeman_pattern(lower, upper):
    """lower/upper = (S, L, J). Returns (shift, weight, kind) arrays."""
    cap = 256
    sh, we, ki = np.zeros(cap), np.zeros(cap), np.zeros(cap, dtype=np.int32)
    n = lib().orc_zeeman_pattern(*[C.c_double(x) for x in (*lower, *upper)], C.c_int(cap),
                                 _p(sh, C.c_double), _p(we, C.c_double), _p(ki, C.c_int))
    return sh[:n].copy(), we[:n].copy(), ki[:n].copy()


class Lines:
    """Line list for the oracle: list of dicts {lambda0, strength, shift[], weight[], kind[]} + lambda_ref."""

    def __init__(self, lines, lambda_ref):
        self.n = len(lines)
        self.lambda_ref = float(lambda_ref)
        self.lambda0 = _f64([l["lambda0"] for l in lines])
        self.strength = _f64([l["strength"] for l in lines])
        self.n_comp = _i32([len(l["shift"]) for l in lines])
        self.shift = _f64(np.concatenate([np.asarray(l["shift"], dtype=np.float64) for l in lines]))
        self.weight = _f64(np.concatenate([np.asarray(l["weight"], dtype=np.float64) for l in lines]))
        self.kind = _i32(np.concatenate([np.asarray(l["kind"], dtype=np.int32) for l in lines]))

    def args(self):
        return [C.c_int(self.n), _p(self.lambda0, C.c_double), _p(self.strength, C.c_double), _p(self.n_comp, C.c_int),
                _p(self.shift, C.c_double), _p(self.weight, C.c_double), _p(self.kind, C.c_int), C.c_double(self.lambda_ref)]


def _npar(cfg):
    return int(len(cfg["lo"]))


def _variant(cfg):
    """0 = real-coded operators (readings G1-G3), 1 = the paper's binary-coded GA (readings V0-V5)."""
    return int(cfg.get("variant", 0))


def prologue(obs, cfg):
    """obs[N,4,L] -> [N,6]: w_I, w_Q, w_U, w_V (eq. 20-23) and the inclination box, per cfg["prologue"] bits."""
    obs = _f64(obs)
    N, L = obs.shape[0], obs.shape[2]
    w, sg = _f64(cfg["stokes_weight"]), _f64(cfg["sigma"])
    out = np.empty((N, 6))
    lib().orc_prologue(_p(obs, C.c_double), C.c_int64(N), C.c_int(L), _p(w, C.c_double), _p(sg, C.c_double),
                       C.c_double(cfg["lo"][1]), C.c_double(cfg["hi"][1]), C.c_int(int(cfg.get("prologue", 0))), _p(out, C.c_double))
    return out


def uncertainty_step():
    """The finite-difference step h of reading U1, in box coordinates."""
    f = lib().orc_uncertainty_step
    f.restype = C.c_double
    return float(f())


def uncertainty(obs, params, lam, lines, cfg, mu=None, nm_profile=None, threads=1, want_hessian=False):
    """eq. 26 / reading U1: obs[N,4,L], params[N,M] (the optimum) -> (sigma[N,M], chi2[N]) and, if asked, the Hessians
    [N,M,M] in box coordinates."""
    obs, lam, params = _f64(obs), _f64(lam), _f64(params)
    N, L, npar = obs.shape[0], lam.size, _npar(cfg)
    assert params.shape == (N, npar)
    mu_a = _f64(mu) if mu is not None else None
    nm = _nm(nm_profile, npar, L)
    lo, hi, lg = _f64(cfg["lo"]), _f64(cfg["hi"]), _i32(cfg["log_scale"])
    w, sg = _f64(cfg["stokes_weight"]), _f64(cfg["sigma"])
    sig, chi = np.empty((N, npar)), np.empty(N)
    hess = np.empty((N, npar, npar)) if want_hessian else None
    lib().orc_uncertainty(_p(obs, C.c_double), _p(mu_a, C.c_double), C.c_int64(N), _p(lam, C.c_double), C.c_int(L),
                          *lines.args(), _p(lo, C.c_double), _p(hi, C.c_double), _p(lg, C.c_int), _p(w, C.c_double),
                          _p(sg, C.c_double), C.c_int(npar), C.c_int(int(cfg.get("prologue", 0))), _p(nm, C.c_double),
                          _p(params, C.c_double), C.c_int(threads), _p(sig, C.c_double), _p(chi, C.c_double),
                          _p(hess, C.c_double))
    return (sig, chi, hess) if want_hessian else (sig, chi)


def uncertainty_n_eval(M):
    return int(lib().orc_uncertainty_n_eval(C.c_int(M)))


def uncertainty_offsets(M, e, h):
    du = np.zeros(M)
    lib().orc_uncertainty_offsets(C.c_int(M), C.c_int(e), C.c_double(h), _p(du, C.c_double))
    return du


def uncertainty_from_chi2(chi2v, M, h, active=None):
    chi2v = _f64(chi2v)
    act = _i32(np.ones(M) if active is None else active)
    out = np.empty(M)
    lib().orc_uncertainty_from_chi2(_p(chi2v, C.c_double), C.c_int(M), C.c_double(h), _p(act, C.c_int), _p(out, C.c_double))
    return out


def seeds(obs, lam, lines, cfg):
    """Reading S1: obs[N,4,L] -> [N,3] = centre-of-gravity B_los [G], and the 10-bit box coordinates (q_B, q_gamma) of the seed."""
    obs, lam = _f64(obs), _f64(lam)
    N, L = obs.shape[0], lam.size
    out = np.empty((N, 3))
    lib().orc_seeds(_p(obs, C.c_double), C.c_int64(N), _p(lam, C.c_double), C.c_int(L), *lines.args(),
                    C.c_double(cfg["lo"][0]), C.c_double(cfg["hi"][0]), C.c_int(int(cfg["log_scale"][0])), _p(out, C.c_double))
    return out


def seed_auer(obs, lam, lines, cfg, glo=None, ghi=None):
    """Reading S2: obs[N,4,L] -> [N,7] = B_los [G], gamma, chi [deg], B [G], and the 10-bit box coordinates (q_B, q_gamma, q_chi)
    of the Auer weak-field member; glo/ghi[N] = per-pixel inclination box (default: the configured one)."""
    obs, lam = _f64(obs), _f64(lam)
    N, L = obs.shape[0], lam.size
    glo = np.full(N, float(cfg["lo"][1])) if glo is None else _f64(glo)
    ghi = np.full(N, float(cfg["hi"][1])) if ghi is None else _f64(ghi)
    out = np.empty((N, 7))
    lib().orc_seed_auer(_p(obs, C.c_double), C.c_int64(N), _p(lam, C.c_double), C.c_int(L), *lines.args(),
                        C.c_double(cfg["lo"][0]), C.c_double(cfg["hi"][0]), C.c_int(int(cfg["log_scale"][0])),
                        C.c_double(cfg["lo"][2]), C.c_double(cfg["hi"][2]), _p(glo, C.c_double), _p(ghi, C.c_double), _p(out, C.c_double))
    return out


def sobol(n0, count, dims):
    out = np.zeros((count, dims), dtype=np.uint32)
    lib().orc_sobol(C.c_uint32(n0), C.c_int(count), C.c_int(dims), _p(out, C.c_uint32))
    return out


def _nm(nm_profile, npar, L):
    if npar == NPAR:
        return None
    assert npar == 11 and nm_profile is not None, "the 11-parameter model needs nm_profile[L] (reading F13)"
    a = _f64(nm_profile)
    assert a.shape == (L,)
    return a


def synth(params, lam, lines, mu=None, use_solve=False, threads=1, nm_profile=None):
    """params[P,9], or [P,11] with nm_profile[L] (11-parameter model, reading F13)."""
    params = _f64(params)
    npar = params.shape[-1] if params.ndim > 1 else params.size
    assert npar in (9, 11)
    params = params.reshape(-1, npar)
    lam = _f64(lam)
    P, L = params.shape[0], lam.size
    mu_a = _f64(mu) if mu is not None else None
    nm = _nm(nm_profile, npar, L)
    out = np.empty((P, 4, L))
    lib().orc_synth(_p(params, C.c_double), C.c_int(npar), _p(nm, C.c_double), _p(mu_a, C.c_double), C.c_int64(P), _p(lam, C.c_double), C.c_int(L),
                    *lines.args(), C.c_int(int(use_solve)), C.c_int(threads), _p(out, C.c_double))
    return out


def absorption_matrix(p, lam, lines):
    p = _f64(p)
    out = np.empty(7)
    lib().orc_absorption_matrix(_p(p, C.c_double), C.c_double(lam), *lines.args(), _p(out, C.c_double))
    return out


def chi2(obs, model, w, sigma, M=NPAR):
    obs, model, w, sigma = _f64(obs), _f64(model), _f64(w), _f64(sigma)
    L = obs.shape[-1]
    return lib().orc_chi2(_p(obs, C.c_double), _p(model, C.c_double), C.c_int(L), _p(w, C.c_double), _p(sigma, C.c_double), C.c_int(M))


def philox(seed, c0, c1, c2, c3):
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(C.c_uint64(seed), C.c_uint32(c0), C.c_uint32(c1), C.c_uint32(c2), C.c_uint32(c3), _p(out, C.c_uint32))
    return out


def philox_raw(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox_raw(_p(ctr, C.c_uint32), _p(key, C.c_uint32), _p(out, C.c_uint32))
    return out


def decode(genes, cfg):
    npar = _npar(cfg)
    genes = np.ascontiguousarray(genes, dtype=np.float32).reshape(-1, npar)
    out = np.empty(genes.shape)
    lo, hi, lg = _f64(cfg["lo"]), _f64(cfg["hi"]), _i32(cfg["log_scale"])
    lib().orc_decode(_p(genes, C.c_float), C.c_int(npar), C.c_int(_variant(cfg)), C.c_int64(genes.shape[0]), _p(lo, C.c_double), _p(hi, C.c_double), _p(lg, C.c_int), _p(out, C.c_double))
    return out


def ga_init(N, pop, seed, pixel_base=0, npar=NPAR, variant=0):
    genes = np.empty((N, pop, npar), dtype=np.float32)
    lib().orc_ga_init(C.c_int64(N), C.c_uint64(pixel_base), C.c_int(pop), C.c_int(npar), C.c_int(variant), C.c_uint64(seed), _p(genes, C.c_float))
    return genes


def _cfg_args(cfg):
    ms = np.ascontiguousarray(cfg["mut_scale"], dtype=np.float32)
    assert ms.size == cfg["generations"] + 1
    keep = [ms]
    return keep, [C.c_int(cfg["pop"]), C.c_int(cfg["generations"]), C.c_int(cfg["tournament_k"]),
                  C.c_float(cfg["p_cross"]), C.c_float(cfg["p_mut"]), _p(ms, C.c_float)]


def ga_step(genes, chi2v, t, cfg, seed, pixel_base=0):
    genes = np.ascontiguousarray(genes, dtype=np.float32)
    N, pop = genes.shape[0], genes.shape[1]
    chi2v = _f64(chi2v)
    out = np.empty_like(genes)
    keep, a = _cfg_args(cfg)
    per = _i32(cfg["periodic"])
    lib().orc_ga_step(_p(genes, C.c_float), _p(chi2v, C.c_double), C.c_int64(N), C.c_uint64(pixel_base), C.c_int(t),
                      *a, _p(per, C.c_int), C.c_int(genes.shape[2]), C.c_int(_variant(cfg)), C.c_uint64(seed), _p(out, C.c_float))
    return out


def ga_fitness(genes, obs, lam, lines, cfg, mu=None, threads=1, nm_profile=None):
    genes = np.ascontiguousarray(genes, dtype=np.float32)
    N, pop = genes.shape[0], genes.shape[1]
    obs, lam = _f64(obs), _f64(lam)
    mu_a = _f64(mu) if mu is not None else None
    lo, hi, lg = _f64(cfg["lo"]), _f64(cfg["hi"]), _i32(cfg["log_scale"])
    w, sg = _f64(cfg["stokes_weight"]), _f64(cfg["sigma"])
    npar = _npar(cfg)
    assert genes.shape[2] == npar
    nm = _nm(nm_profile, npar, lam.size)
    out = np.empty((N, pop))
    lib().orc_ga_fitness(_p(genes, C.c_float), _p(obs, C.c_double), _p(mu_a, C.c_double), C.c_int64(N), C.c_int(pop),
                         _p(lam, C.c_double), C.c_int(lam.size), *lines.args(),
                         _p(lo, C.c_double), _p(hi, C.c_double), _p(lg, C.c_int), _p(w, C.c_double), _p(sg, C.c_double),
                         C.c_int(npar), C.c_int(_variant(cfg)), _p(nm, C.c_double), C.c_int(threads), _p(out, C.c_double))
    return out


def ga_invert(obs, lam, lines, cfg, seed, mask=None, mu=None, pixel_base=0, threads=1, want_trace=False, nm_profile=None):
    """obs[N,4,L] -> dict(params[N,M], chi2[N], genes[N,M], trace[N,G+1] or None); M = len(cfg["lo"]) = 9 or 11."""
    obs, lam = _f64(obs), _f64(lam)
    N, L = obs.shape[0], lam.size
    assert obs.shape == (N, 4, L)
    mu_a = _f64(mu) if mu is not None else None
    mask_a = np.ascontiguousarray(mask, dtype=np.uint8) if mask is not None else None
    lo, hi, lg, per = _f64(cfg["lo"]), _f64(cfg["hi"]), _i32(cfg["log_scale"]), _i32(cfg["periodic"])
    w, sg = _f64(cfg["stokes_weight"]), _f64(cfg["sigma"])
    keep, a = _cfg_args(cfg)
    npar = _npar(cfg)
    nm = _nm(nm_profile, npar, L)
    params, chi2v = np.empty((N, npar)), np.empty(N)
    genes = np.full((N, npar), np.nan, dtype=np.float32)
    trace = np.full((N, cfg["generations"] + 1), np.nan) if want_trace else None
    lib().orc_ga_invert(_p(obs, C.c_double), _p(mask_a, C.c_ubyte), _p(mu_a, C.c_double), C.c_int64(N), C.c_uint64(pixel_base),
                        _p(lam, C.c_double), C.c_int(L), *lines.args(), *a,
                        _p(lo, C.c_double), _p(hi, C.c_double), _p(lg, C.c_int), _p(per, C.c_int),
                        _p(w, C.c_double), _p(sg, C.c_double), C.c_int(npar), C.c_int(_variant(cfg)), C.c_int(int(cfg.get("prologue", 0))), _p(nm, C.c_double), C.c_uint64(seed), C.c_int(threads),
                        _p(params, C.c_double), _p(chi2v, C.c_double), _p(genes, C.c_float), _p(trace, C.c_double))
    return {"params": params, "chi2": chi2v, "genes": genes, "trace": trace}
