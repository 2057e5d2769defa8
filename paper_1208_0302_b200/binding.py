"""Thin Python binding over the C ABI of include/me.h (libme_b200.so): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  torch is used for device memory and streams.
There is no CPU fallback: importing works without a GPU (so that symbols can be checked), but every compute call
raises if the library or a CUDA device is missing.
"""
import ctypes as C
import os

import numpy as np

NPAR = 9
MAX_NPAR = 11      # with fill fraction and stray-light fraction (include/me.h ME_MAX_NPAR)
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libme_b200.so")
_lib = None

EXPORTS = ["me_synth", "me_synth_ws", "me_synth_workspace_bytes", "me_synth_static", "me_synth_static_max_vectors", "ga_invert", "ga_uncertainty", "ga_step", "ga_fitness", "ga_init", "ga_prologue", "me_philox", "me_philox_many", "me_faddeeva",
           "me_zeeman_pattern", "me_peak_probe", "me_strerror", "me_last_cuda_error", "me_version"]


class MeError(RuntimeError):
    def __init__(self, code, where):
        l = lib()
        msg = l.me_strerror(code).decode()
        if code == -5:
            msg += ": " + l.me_last_cuda_error().decode()
        super().__init__("%s failed with %d (%s)" % (where, code, msg))
        self.code = code


class _MeLine(C.Structure):
    _fields_ = [("lambda0_A", C.c_double), ("strength", C.c_float), ("n_comp", C.c_int),
                ("shift", C.POINTER(C.c_float)), ("weight", C.POINTER(C.c_float)), ("kind", C.POINTER(C.c_int8))]


class _MeLineData(C.Structure):
    _fields_ = [("n_lines", C.c_int), ("lines", C.POINTER(_MeLine)), ("lambda_ref_A", C.c_double),
                ("n_params", C.c_int), ("nm_profile", C.c_void_p)]


class _GaCfg(C.Structure):
    _fields_ = [("pop", C.c_int), ("generations", C.c_int), ("tournament_k", C.c_int), ("elite", C.c_int),
                ("p_cross", C.c_float), ("p_mut", C.c_float), ("mut_scale0", C.c_float), ("mut_scale_end", C.c_float),
                ("mut_scale_table", C.POINTER(C.c_float)),
                ("lo", C.c_float * MAX_NPAR), ("hi", C.c_float * MAX_NPAR),
                ("log_scale", C.c_uint8 * MAX_NPAR), ("periodic", C.c_uint8 * MAX_NPAR),
                ("stokes_weight", C.c_float * 4), ("mu", C.c_void_p), ("pixel_id_base", C.c_int64),
                ("variant", C.c_int), ("prologue", C.c_int)]


def lib():
    """Loads libme_b200.so; fails loudly if it has not been built (python -m paper_1208_0302_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libme_b200.so is missing: run `python -m paper_1208_0302_b200.build` (nvcc, sm_100a). "
                               "There is no CPU fallback.")
        l = C.CDLL(LIB_PATH)
        l.me_strerror.restype = C.c_char_p
        l.me_last_cuda_error.restype = C.c_char_p
        l.me_strerror.argtypes = [C.c_int]
        l.me_synth_workspace_bytes.restype = C.c_size_t
        l.me_synth_workspace_bytes.argtypes = [C.c_int64]
        l.me_synth_static_max_vectors.restype = C.c_int64
        l.me_synth_static_max_vectors.argtypes = []
        _lib = l
    return _lib


def _check(code, where):
    if code != 0:
        raise MeError(code, where)


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, dtype, name):
    import torch
    if t is None:
        return C.c_void_p(0)
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return C.c_void_p(t.data_ptr())


class LineData:
    """Host-side line list. lines: list of dict(lambda0, strength, shift[], weight[], kind[])."""

    def __init__(self, lines, lambda_ref, n_params=NPAR, nm_profile=None):
        """n_params = 11 needs nm_profile: a contiguous CUDA f32 tensor [L] (I_fixed, reading F13)."""
        self._keep = [nm_profile]
        self.n_params = int(n_params)
        arr = (_MeLine * len(lines))()
        for i, l in enumerate(lines):
            sh = np.ascontiguousarray(l["shift"], dtype=np.float32)
            we = np.ascontiguousarray(l["weight"], dtype=np.float32)
            ki = np.ascontiguousarray(l["kind"], dtype=np.int8)
            self._keep += [sh, we, ki]
            arr[i] = _MeLine(float(l["lambda0"]), float(l["strength"]), int(sh.size),
                             sh.ctypes.data_as(C.POINTER(C.c_float)), we.ctypes.data_as(C.POINTER(C.c_float)),
                             ki.ctypes.data_as(C.POINTER(C.c_int8)))
        self._arr = arr
        nm_ptr = None
        if nm_profile is not None:
            import torch
            nm_ptr = _dev(nm_profile, torch.float32, "nm_profile").value
        self.c = _MeLineData(len(lines), arr, float(lambda_ref), int(n_params), nm_ptr)


def zeeman_pattern(lower, upper):
    """me_zeeman_pattern: (S,L,J) lower/upper -> (shift, weight, kind) arrays (host-only call)."""
    cap = 256
    sh, we, ki = np.zeros(cap, np.float32), np.zeros(cap, np.float32), np.zeros(cap, np.int8)
    n = lib().me_zeeman_pattern(*[C.c_double(x) for x in (*lower, *upper)], C.c_int(cap),
                                sh.ctypes.data_as(C.POINTER(C.c_float)), we.ctypes.data_as(C.POINTER(C.c_float)),
                                ki.ctypes.data_as(C.POINTER(C.c_int8)))
    if n < 0:
        raise MeError(n, "me_zeeman_pattern")
    return sh[:n].copy(), we[:n].copy(), ki[:n].copy()


def line_data_from_workload(lines, triplets=True, lambda_ref=None, n_params=NPAR, nm_profile=None):
    """Builds a LineData from workloads.FE_* dicts: effective triplets, or the full pattern via me_zeeman_pattern."""
    from . import workloads as W
    out = []
    for l in lines:
        if triplets:
            g = l["g_eff"]
            sh, we, ki = [0.0, -g, g], [1.0, 1.0, 1.0], [0, -1, 1]
        else:
            sh, we, ki = zeeman_pattern(l["lower"], l["upper"])
        out.append(dict(lambda0=l["lambda0"], strength=l["strength"], shift=sh, weight=we, kind=ki))
    return LineData(out, W.LAMBDA_REF if lambda_ref is None else lambda_ref, n_params, nm_profile)


def make_ga_cfg(cfg, mu=None, pixel_id_base=0):
    """cfg: dict from workloads.ga_config. Returns (_GaCfg, keepalive)."""
    ms = np.ascontiguousarray(cfg["mut_scale"], dtype=np.float32)
    assert ms.size == cfg["generations"] + 1
    c = _GaCfg()
    c.pop, c.generations, c.tournament_k, c.elite = cfg["pop"], cfg["generations"], cfg["tournament_k"], 1
    c.p_cross, c.p_mut = cfg["p_cross"], cfg["p_mut"]
    c.mut_scale0, c.mut_scale_end = float(ms[0]), float(ms[-1])
    c.mut_scale_table = ms.ctypes.data_as(C.POINTER(C.c_float))
    for j in range(len(cfg["lo"])):
        c.lo[j], c.hi[j] = float(cfg["lo"][j]), float(cfg["hi"][j])
        c.log_scale[j], c.periodic[j] = int(cfg["log_scale"][j]), int(cfg["periodic"][j])
    for s in range(4):
        c.stokes_weight[s] = float(cfg["stokes_weight"][s])
    import torch
    c.mu = _dev(mu, torch.float32, "mu").value if mu is not None else None
    c.pixel_id_base = int(pixel_id_base)
    c.variant = int(cfg.get("variant", 0))
    c.prologue = int(cfg.get("prologue", 0))
    return c, (ms, mu)


def _grid(lam):
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    return lam, lam.ctypes.data_as(C.POINTER(C.c_double)), C.c_int(lam.size)


def me_synth_workspace_bytes(P):
    return int(lib().me_synth_workspace_bytes(C.c_int64(P)))


def me_synth(params, lam, line_data, mu=None, out_stokes=None, obs_ref=None, w_over_sigma=None, out_chi2=None, want_stokes=True,
             workspace=None):
    """params: CUDA f32 [P, line_data.n_params]. Returns (out_stokes [P,4,L] or None, out_chi2 [P] or None).

    workspace: a CUDA uint8 tensor of >= me_synth_workspace_bytes(P) bytes for the ordered visit of large batches (me_synth_ws);
    None = allocate one here from torch's caching allocator when the library asks for one; False = none (plain me_synth)."""
    import torch
    P = params.shape[0]
    assert params.dim() == 2 and params.shape[1] == line_data.n_params
    lam, lam_p, L = _grid(lam)
    if out_stokes is None and want_stokes:
        out_stokes = torch.empty((P, 4, lam.size), dtype=torch.float32, device=params.device)
    wos = None
    if obs_ref is not None:
        wos = np.ascontiguousarray(w_over_sigma, dtype=np.float32)
        if out_chi2 is None:
            out_chi2 = torch.empty((P,), dtype=torch.float32, device=params.device)
    if workspace is None:
        need = me_synth_workspace_bytes(P)
        workspace = torch.empty((need,), dtype=torch.uint8, device=params.device) if need else False
    ws_bytes = 0 if workspace is False else int(workspace.numel())
    _check(lib().me_synth_ws(_dev(params, torch.float32, "params"), C.c_int64(P), _dev(mu, torch.float32, "mu"), lam_p, L,
                             C.byref(line_data.c), _dev(out_stokes, torch.float32, "out_stokes"),
                             _dev(obs_ref, torch.float32, "obs_ref"),
                             wos.ctypes.data_as(C.POINTER(C.c_float)) if wos is not None else None,
                             _dev(out_chi2, torch.float32, "out_chi2"),
                             _dev(None if workspace is False else workspace, torch.uint8, "workspace"), C.c_size_t(ws_bytes),
                             _stream()), "me_synth_ws")
    return out_stokes, out_chi2


def me_synth_static_max_vectors():
    return int(lib().me_synth_static_max_vectors())


def me_synth_static(params, lam, line_data, mu=None, out_stokes=None, obs_ref=None, w_over_sigma=None, out_chi2=None):
    """me_synth through the entry point that allocates nothing: the ordering scratch is the library's fixed device array
    (include/me.h).  out_stokes [P,4,L] is the CALLER's (required; pass out_chi2 too if chi2 is wanted): nothing is allocated
    here either.  Returns (out_stokes, out_chi2)."""
    import torch
    P = params.shape[0]
    assert params.dim() == 2 and params.shape[1] == line_data.n_params
    lam, lam_p, L = _grid(lam)
    assert out_stokes is not None or out_chi2 is not None, "the caller passes the outputs"
    wos = np.ascontiguousarray(w_over_sigma, dtype=np.float32) if obs_ref is not None else None
    _check(lib().me_synth_static(_dev(params, torch.float32, "params"), C.c_int64(P), _dev(mu, torch.float32, "mu"), lam_p, L,
                                 C.byref(line_data.c), _dev(out_stokes, torch.float32, "out_stokes"),
                                 _dev(obs_ref, torch.float32, "obs_ref"),
                                 wos.ctypes.data_as(C.POINTER(C.c_float)) if wos is not None else None,
                                 _dev(out_chi2, torch.float32, "out_chi2"), _stream()), "me_synth_static")
    return out_stokes, out_chi2


def ga_invert(obs, lam, line_data, cfg, seed, mask=None, mu=None, pixel_id_base=0, out_params=None, out_chi2=None):
    """obs: CUDA f32 [N,4,L]. Returns (out_params [N, n_params], out_chi2 [N])."""
    import torch
    N = obs.shape[0]
    lam, lam_p, L = _grid(lam)
    assert tuple(obs.shape) == (N, 4, lam.size)
    assert len(cfg["lo"]) == line_data.n_params
    c, keep = make_ga_cfg(cfg, mu, pixel_id_base)
    sig = np.ascontiguousarray(cfg["sigma"], dtype=np.float32)
    if out_params is None:
        out_params = torch.empty((N, line_data.n_params), dtype=torch.float32, device=obs.device)
    if out_chi2 is None:
        out_chi2 = torch.empty((N,), dtype=torch.float32, device=obs.device)
    _check(lib().ga_invert(_dev(obs, torch.float32, "obs"), C.c_int64(N), _dev(mask, torch.uint8, "mask"),
                           sig.ctypes.data_as(C.POINTER(C.c_float)), lam_p, L, C.byref(line_data.c), C.byref(c),
                           C.c_uint64(seed), _dev(out_params, torch.float32, "out_params"),
                           _dev(out_chi2, torch.float32, "out_chi2"), _stream()), "ga_invert")
    return out_params, out_chi2


def ga_fitness(genes, obs, lam, line_data, cfg, mu=None):
    import torch
    N, pop = genes.shape[0], genes.shape[1]
    lam, lam_p, L = _grid(lam)
    c, keep = make_ga_cfg(cfg, mu)
    assert pop == cfg["pop"] and genes.shape[2] == line_data.n_params == len(cfg["lo"])
    sig = np.ascontiguousarray(cfg["sigma"], dtype=np.float32)
    out = torch.empty((N, pop), dtype=torch.float32, device=genes.device)
    _check(lib().ga_fitness(_dev(genes, torch.float32, "genes"), _dev(obs, torch.float32, "obs"), C.c_int64(N),
                            sig.ctypes.data_as(C.POINTER(C.c_float)), lam_p, L, C.byref(line_data.c), C.byref(c),
                            _dev(out, torch.float32, "chi2_out"), _stream()), "ga_fitness")
    return out


def ga_step(genes, chi2, t, cfg, seed, pixel_id_base=0):
    import torch
    N, pop = genes.shape[0], genes.shape[1]
    assert pop == cfg["pop"]
    c, keep = make_ga_cfg(cfg, None, pixel_id_base)
    out = torch.empty_like(genes)
    _check(lib().ga_step(_dev(genes, torch.float32, "genes_in"), _dev(chi2, torch.float32, "chi2_in"), C.c_int64(N),
                         C.c_int(t), C.byref(c), C.c_int(genes.shape[2]), C.c_uint64(seed), _dev(out, torch.float32, "genes_out"),
                         _stream()), "ga_step")
    return out


def ga_init(N, cfg, seed, pixel_id_base=0, device="cuda"):
    import torch
    c, keep = make_ga_cfg(cfg, None, pixel_id_base)
    npar = len(cfg["lo"])
    out = torch.empty((N, cfg["pop"], npar), dtype=torch.float32, device=device)
    _check(lib().ga_init(C.c_int64(N), C.byref(c), C.c_int(npar), C.c_uint64(seed), _dev(out, torch.float32, "genes_out"), _stream()), "ga_init")
    return out


def me_philox(seed, c0, c1, c2, c3):
    out = (C.c_uint32 * 4)()
    _check(lib().me_philox(C.c_uint64(seed), C.c_uint32(c0), C.c_uint32(c1), C.c_uint32(c2), C.c_uint32(c3), out), "me_philox")
    return np.array(list(out), dtype=np.uint32)


def me_philox_many(seed, c0_base, c1, c2, c3, n, device="cuda"):
    import torch
    out = torch.empty((n, 4), dtype=torch.int32, device=device)
    _check(lib().me_philox_many(C.c_uint64(seed), C.c_uint32(c0_base), C.c_uint32(c1), C.c_uint32(c2), C.c_uint32(c3),
                                C.c_int64(n), C.c_void_p(out.data_ptr()), _stream()), "me_philox_many")
    return out


def me_faddeeva(v, a):
    import torch
    H, F = torch.empty_like(v), torch.empty_like(v)
    _check(lib().me_faddeeva(_dev(v, torch.float32, "v"), _dev(a, torch.float32, "a"), C.c_int64(v.numel()),
                             _dev(H, torch.float32, "H"), _dev(F, torch.float32, "F"), _stream()), "me_faddeeva")
    return H, F


def me_peak_probe(kind, iters, blocks, scratch):
    """Launches one instruction-throughput probe (see include/me.h); returns the lane-slot count it executes."""
    import torch
    assert scratch.numel() >= blocks * 256
    _check(lib().me_peak_probe(C.c_int(kind), C.c_int(iters), C.c_int(blocks), _dev(scratch, torch.float32, "out"), _stream()),
           "me_peak_probe")
    return blocks * 256 * iters * 32


def ga_prologue(obs, lam, line_data, cfg):
    """obs: CUDA f32 [N,4,L]. Returns [N,12]: w_I, w_Q, w_U, w_V, gamma_lo, gamma_hi as ga_invert uses them, then B_los [G] and
    the stored genes (B, gamma) of the centre-of-gravity member, then the stored genes (B, gamma, chi) of the Auer weak-field
    member (cfg["prologue"] bit flags 4 and 8)."""
    import torch
    N = obs.shape[0]
    lam, lam_p, L = _grid(lam)
    c, keep = make_ga_cfg(cfg)
    sig = np.ascontiguousarray(cfg["sigma"], dtype=np.float32)
    out = torch.empty((N, 12), dtype=torch.float32, device=obs.device)
    _check(lib().ga_prologue(_dev(obs, torch.float32, "obs"), C.c_int64(N), sig.ctypes.data_as(C.POINTER(C.c_float)), lam_p, L,
                             C.byref(line_data.c), C.byref(c), _dev(out, torch.float32, "out"), _stream()), "ga_prologue")
    return out


def ga_uncertainty(obs, params, lam, line_data, cfg, mask=None, mu=None):
    """obs: CUDA f32 [N,4,L]; params: CUDA f32 [N,M] (the optimum). Returns (sigma [N,M], chi2 [N]) per eq. 26."""
    import torch
    N = obs.shape[0]
    lam, lam_p, L = _grid(lam)
    assert tuple(params.shape) == (N, line_data.n_params) and len(cfg["lo"]) == line_data.n_params
    c, keep = make_ga_cfg(cfg, mu)
    sig = np.ascontiguousarray(cfg["sigma"], dtype=np.float32)
    out_s = torch.empty((N, line_data.n_params), dtype=torch.float32, device=obs.device)
    out_c = torch.empty((N,), dtype=torch.float32, device=obs.device)
    _check(lib().ga_uncertainty(_dev(obs, torch.float32, "obs"), C.c_int64(N), _dev(mask, torch.uint8, "mask"),
                                sig.ctypes.data_as(C.POINTER(C.c_float)), lam_p, L, C.byref(line_data.c), C.byref(c),
                                _dev(params, torch.float32, "params"), _dev(out_s, torch.float32, "out_sigma"),
                                _dev(out_c, torch.float32, "out_chi2"), _stream()), "ga_uncertainty")
    return out_s, out_c
