"""No-GPU checks of the C-ABI library: it loads, exports every symbol include/me.h declares, validates arguments
(no compute call is made), and its host-only Zeeman helper agrees with Table 1 and with the oracle's."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1208_0302_b200 import binding as B
from paper_1208_0302_b200 import build as mebuild
from paper_1208_0302_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    mebuild.build()
    return B.lib()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "me.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"^\s*(?:const\s+char\s*\*|int|int64_t|size_t)\s+(\w+)\s*\(", hdr, flags=re.M))
    assert {"me_synth", "ga_invert", "ga_step", "ga_fitness", "me_philox"} <= names
    assert names == set(B.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n
    assert lib.me_version() >= 100
    assert lib.me_strerror(-3) == b"a value is out of range"


def test_struct_layout_matches_header(lib):
    # sizes the C compiler gives for the header's structs must equal the ctypes mirrors
    import subprocess, tempfile
    src = '#include "me.h"\n#include <stdio.h>\nint main(){printf("%zu %zu %zu\\n", sizeof(me_line), sizeof(me_line_data), sizeof(ga_cfg));return 0;}'
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "s.c"), "w").write(src)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(d, "s"), os.path.join(d, "s.c")], check=True)
        out = subprocess.run([os.path.join(d, "s")], capture_output=True, text=True, check=True).stdout.split()
    assert [int(x) for x in out] == [C.sizeof(B._MeLine), C.sizeof(B._MeLineData), C.sizeof(B._GaCfg)]


def test_zeeman_helper_table1_and_oracle(lib):
    from oracle import api as orc
    sh, we, ki = B.zeeman_pattern(W.FE_6301["lower"], W.FE_6301["upper"])
    assert len(sh) == 12
    assert abs((we[ki == 1] * sh[ki == 1]).sum() - 5 / 3) < 1e-6        # Table 1: g_eff = 1.667
    sh2, we2, ki2 = B.zeeman_pattern(W.FE_6302["lower"], W.FE_6302["upper"])
    assert sorted(zip(ki2.tolist(), sh2.tolist(), we2.tolist())) == [(-1, -2.5, 1.0), (0, 0.0, 1.0), (1, 2.5, 1.0)]
    for lo, up in [((2, 1, 2), (2, 2, 2)), ((1, 2, 3), (1, 3, 4)), ((1.5, 2, 3.5), (1.5, 1, 2.5)), ((0, 0, 0), (0, 1, 1))]:
        a = sorted(zip(*[x.tolist() for x in B.zeeman_pattern(lo, up)][::-1]))
        b = sorted(zip(*[x.tolist() for x in orc.zeeman_pattern(lo, up)][::-1]))
        assert len(a) == len(b)
        assert np.allclose(np.array(a, dtype=float), np.array(b, dtype=float), atol=1e-6)
    assert lib.me_zeeman_pattern(C.c_double(0), C.c_double(0), C.c_double(0), C.c_double(0), C.c_double(0), C.c_double(0),
                                 0, None, None, None) == -3     # J = 0 -> J = 0 is forbidden


def _cfg_ld():
    c0 = W.config0()
    ld = B.line_data_from_workload(c0["lines"], True)
    return c0, ld


def test_argument_validation_without_gpu(lib):
    c0, ld = _cfg_ld()
    lam = np.ascontiguousarray(c0["lam"])
    lam_p = lam.ctypes.data_as(C.POINTER(C.c_double))
    sig = (C.c_float * 4)(1e-3, 1e-3, 1e-3, 1e-3)
    cfg, keep = None, None
    import unittest.mock as um
    with um.patch.object(B, "_dev", lambda t, d, n: C.c_void_p(0)):
        cfg, keep = B.make_ga_cfg(c0["ga"])
    one = C.c_void_p(16)     # non-null dummy; never dereferenced because validation fails first or N == 0
    call = lambda **kw: lib.ga_invert(kw.get("obs", one), C.c_int64(kw.get("N", 4)), None, kw.get("sigma", sig),
                                      kw.get("lam", lam_p), C.c_int(kw.get("L", lam.size)), C.byref(kw.get("ld", ld.c)),
                                      C.byref(kw.get("cfg", cfg)), C.c_uint64(1),
                                      kw.get("outp", one), one, None)
    assert call(N=0) == 0                                      # empty input is a no-op
    assert call(obs=None) == -1
    assert call(lam=None) == -1
    assert call(L=1) == -2 and call(L=513) == -2
    assert call(sigma=None) == -1
    assert call(sigma=(C.c_float * 4)(1e-3, 0.0, 1e-3, 1e-3)) == -3
    bad = B._GaCfg.from_buffer_copy(cfg); bad.pop = 1
    assert call(cfg=bad) == -2
    bad = B._GaCfg.from_buffer_copy(cfg); bad.pop = 2000
    assert call(cfg=bad) == -2
    bad = B._GaCfg.from_buffer_copy(cfg); bad.lo[3] = 60.0
    assert call(cfg=bad) == -3                                 # lo > hi
    bad = B._GaCfg.from_buffer_copy(cfg); bad.lo[0] = 0.0
    assert call(cfg=bad) == -3                                 # log-scaled gene with lo = 0
    bad = B._GaCfg.from_buffer_copy(cfg); bad.elite = 2
    assert call(cfg=bad) == -4
    bad = B._GaCfg.from_buffer_copy(cfg); bad.pixel_id_base = 2 ** 32 - 2
    assert call(cfg=bad) == -3
    ld11 = B.line_data_from_workload(c0["lines"], True); ld11.c.n_params = 11
    assert call(ld=ld11.c) == -1                               # 11 parameters without the fixed profile (reading F13)
    ld11.c.n_params = 10
    assert call(ld=ld11.c) == -2
    ld9 = B.line_data_from_workload(c0["lines"], True); ld9.c.nm_profile = 16
    assert call(ld=ld9.c) == -2                                # a fixed profile makes no sense with 9 parameters
    # nu = 4 L - M of eq. 16 must be positive: L = 2 gives 8 - 9 < 0 (the argmin compares raw float bits, a negative chi2 breaks it)
    assert call(L=2) == -2
    # the wavelength grid must be finite and strictly increasing (lobe order and centre of gravity of the prologue assume it)
    for bad_lam in (lam[::-1].copy(), np.where(np.arange(lam.size) == 7, np.nan, lam), np.where(np.arange(lam.size) == 7, lam[6], lam)):
        assert call(lam=np.ascontiguousarray(bad_lam).ctypes.data_as(C.POINTER(C.c_double))) == -3
    # reading S1: the seeds take the last two slots of P0, a population of 2 has no room for them
    bad = B._GaCfg.from_buffer_copy(cfg); bad.prologue = 4; bad.pop = 2
    assert call(cfg=bad) == -2
    bad.pop = 3
    assert call(cfg=bad, N=0) == 0
    # ga_uncertainty and ga_prologue ignore the GA fields of cfg (me.h): garbage there is not an error for them ...
    junk = B._GaCfg.from_buffer_copy(cfg)
    junk.pop, junk.generations, junk.tournament_k, junk.elite, junk.p_cross, junk.p_mut = 0, -5, 99, 0, 7.0, -1.0
    junk.mut_scale_table = C.POINTER(C.c_float)(); junk.mut_scale0 = junk.mut_scale_end = 0.0
    assert call(cfg=junk) != 0                                 # ... while ga_invert refuses it
    assert lib.ga_uncertainty(one, C.c_int64(0), None, sig, lam_p, C.c_int(lam.size), C.byref(ld.c), C.byref(junk), one, one, one, None) == 0
    assert lib.ga_prologue(one, C.c_int64(0), sig, lam_p, C.c_int(lam.size), C.byref(ld.c), C.byref(junk), one, None) == 0
    junk.lo[3] = 60.0                                          # their box checks stay
    assert lib.ga_uncertainty(one, C.c_int64(0), None, sig, lam_p, C.c_int(lam.size), C.byref(ld.c), C.byref(junk), one, one, one, None) == -3
    # me_synth
    assert lib.me_synth(one, C.c_int64(0), None, lam_p, C.c_int(lam.size), C.byref(ld.c), one, None, None, None, None) == 0
    assert lib.me_synth(one, C.c_int64(5), None, lam_p, C.c_int(lam.size), C.byref(ld.c), None, None, None, None, None) == -1
    assert lib.me_synth(one, C.c_int64(5), None, lam_p, C.c_int(lam.size), C.byref(ld.c), None, None, None, one, None) == -1
    assert lib.me_synth(one, C.c_int64(-1), None, lam_p, C.c_int(lam.size), C.byref(ld.c), one, None, None, None, None) == -2
    # too many components
    many = [dict(lambda0=6302.0, strength=1.0, shift=np.zeros(30), weight=np.ones(30), kind=np.zeros(30))] * 2
    assert lib.me_synth(one, C.c_int64(0), None, lam_p, C.c_int(lam.size), C.byref(B.LineData(many, 6302.0).c), one, None, None, None, None) == -2


def test_binding_fails_loudly_without_library(monkeypatch):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", "/nonexistent/libme_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.lib()
