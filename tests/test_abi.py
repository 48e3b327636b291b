"""The C-ABI library loads without a GPU and exports every symbol include/psr.h declares; host-side
argument checks that need no device."""
import ctypes as C
import re
from pathlib import Path

import numpy as np

from paper_2005_11468_b200 import binding, synth

ROOT = Path(__file__).resolve().parent.parent


def declared_symbols():
    text = (ROOT / "include" / "psr.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(psr_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    lib = binding.lib()          # dlopen resolves every internal symbol (RTLD_NOW semantics of ctypes)
    syms = declared_symbols()
    assert {"psr_mech_load", "psr_mech_free", "psr_eval_kf_kr", "psr_eval_wdot", "psr_eval_residual",
            "psr_fd_jacobian", "psr_last_error"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s
    assert set(binding.EXPORTS) == set(syms)
    assert b"sm_100a" in lib.psr_version()


def test_mech_load_rejects_malformed_descriptions_before_touching_the_device():
    mech, _ = synth.make_config("C0", 1)
    lib = binding.lib()

    def status(arrays, K=mech.n_species, I=mech.n_reactions):
        desc, keep = binding.make_desc(K, I, arrays)
        h = C.c_void_p()
        st = lib.psr_mech_load(C.byref(desc), C.byref(h))
        assert h.value is None or st == 0
        if st == 0:
            lib.psr_mech_free(h)
        return st, lib.psr_last_error().decode()

    a = mech.arrays()
    bad = dict(a); bad["W"] = a["W"].copy(); bad["W"][3] = 0.0
    assert status(bad)[0] == binding.PSR_EINVAL
    bad = dict(a); bad["reac_sp"] = a["reac_sp"].copy(); bad["reac_sp"][0] = mech.n_species
    st, msg = status(bad); assert st == binding.PSR_EINVAL and "out of range" in msg
    bad = dict(a); bad["reac_nu"] = a["reac_nu"].copy(); bad["reac_nu"][0] = 4
    assert status(bad)[0] == binding.PSR_EINVAL
    bad = dict(a); bad["rtype"] = a["rtype"].copy(); bad["rtype"][0] = 7
    assert status(bad)[0] == binding.PSR_EINVAL
    bad = dict(a); bad["A"] = a["A"].copy(); bad["A"][0] = float("nan")
    st, msg = status(bad); assert st == binding.PSR_EINVAL and "finite" in msg
    bad = dict(a); bad["A"] = a["A"].copy(); bad["A"][0] = float("inf")
    assert status(bad)[0] == binding.PSR_EINVAL
    # any finite A is a valid mechanism: negative and zero pre-exponentials pass validation
    # (without a device the load then stops at PSR_ECUDA, with one it succeeds)
    for v in (-1.0, 0.0):
        ok = dict(a); ok["A"] = a["A"].copy(); ok["A"][0] = v
        assert status(ok)[0] in (binding.PSR_OK, binding.PSR_ECUDA)
    bad = dict(a); bad["nasa"] = None
    assert status(bad)[0] == binding.PSR_EINVAL
    assert status(a, K=0)[0] == binding.PSR_EINVAL
    # Troe parameters: finite, T*** and T* non-zero, T** finite or +inf
    m1, _ = synth.make_config("C1", 1)
    a1 = m1.arrays()
    k = int(np.flatnonzero(np.asarray(a1["rtype"]) == 3)[0])
    def status1(arrs):
        desc, keep = binding.make_desc(m1.n_species, m1.n_reactions, arrs)
        h = C.c_void_p()
        st = lib.psr_mech_load(C.byref(desc), C.byref(h))
        if st == 0:
            lib.psr_mech_free(h)
        return st
    for col, v, want in ((1, 0.0, False), (2, float("nan"), False), (0, float("inf"), False), (3, float("-inf"), False),
                         (3, float("inf"), True)):
        t = dict(a1); t["troe"] = np.array(a1["troe"], dtype=np.float64).copy(); t["troe"][k, col] = v
        st = status1(t)
        assert (st in (binding.PSR_OK, binding.PSR_ECUDA)) if want else st == binding.PSR_EINVAL, (col, v, st)
    assert status(a, K=513)[0] in (binding.PSR_EINVAL, binding.PSR_EUNSUPPORTED)


def test_eval_calls_validate_arguments_without_a_device():
    lib = binding.lib()
    null = C.c_void_p()
    assert lib.psr_eval_wdot(null, 4, null, null, null, 4, null, null, 0, null) == binding.PSR_EINVAL
    assert b"null mechanism" in lib.psr_last_error()
    assert lib.psr_eval_kf_kr(null, -1, null, null, null, 0, null, null, 0, null) == binding.PSR_EINVAL
    assert lib.psr_fd_jacobian(null, 1, null, null, null, null, null, 1, null, null, null) == binding.PSR_EINVAL


def test_solve_calls_validate_arguments_without_a_device():
    lib = binding.lib()
    null = C.c_void_p()
    one = C.c_void_p(8)          # any non-null address: the checks below fail before anything is dereferenced
    assert lib.psr_lu_solve(-1, 4, one, one, one, null) == binding.PSR_EINVAL
    assert lib.psr_lu_solve(3, 0, one, one, one, null) == binding.PSR_EINVAL
    assert lib.psr_lu_solve(3, 4, null, one, one, null) == binding.PSR_EINVAL
    assert lib.psr_lu_solve(0, 4, null, null, null, null) == binding.PSR_OK          # N = 0: nothing to do
    assert lib.psr_ptc_solve(2, 4, one, one, null, one, one, null) == binding.PSR_EINVAL   # null dt
    assert b"psr_ptc_solve" in lib.psr_last_error()
    two = C.c_void_p(16)
    assert lib.psr_ptc_solve(2, 4, one, two, one, two, one, null) == binding.PSR_EINVAL    # dx aliases F
    assert b"alias" in lib.psr_last_error()
    assert lib.psr_ptc_solve(0, 4, null, null, null, null, null, null) == binding.PSR_OK


def test_paper_shaped_config_is_a_batch_of_identical_reactors():
    """P5: the shape of the paper's timing case -- 101 species,
    542 reactions, every reactor at 1800 K, 1 atm, 50 ms, inlet mole fractions 0.15 / 0.18 / 0.67."""
    mech, b = synth.make_config("P5", 7)
    assert (mech.n_species, mech.n_reactions) == (101, 542)
    assert np.all(b.T == 1800.0) and np.all(b.tau == 50e-3) and np.allclose(b.P, 1.01325e6)
    assert np.all(b.Y == b.Y[:, :1]) and np.all(b.Yin == b.Yin[:, :1])
    assert np.allclose(b.Y.sum(axis=0), 1.0, rtol=0, atol=1e-14) and np.all(b.Y > 0)
    x = b.Yin[:, 0] / mech.W
    x /= x.sum()
    assert np.allclose(x[:3], [0.15, 0.18, 0.67], rtol=1e-13) and np.all(x[3:] == 0)
    m2, _ = synth.make_config("P5", 1)
    assert np.array_equal(m2.A, mech.A)                       # seeded: the same mechanism every time
