"""ctypes loader for the CPU oracle (oracle/psr_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2005_11468_b200 (the CUDA path) and the
CUDA path imports nothing from here.  Inputs arrive as plain numpy arrays whose names follow
the mechanism description of SURVEY.md section 8(b).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "psr_oracle.cpp"
_LIB = _HERE / "libpsr_oracle.so"

_MECH_FIELDS = ("W", "nasa", "A", "b", "Ea", "rtype", "reversible", "reac_ptr", "reac_sp", "reac_nu",
                "prod_ptr", "prod_sp", "prod_nu", "eff_ptr", "eff_sp", "eff_val", "A0", "b0", "Ea0", "troe")
_DTYPES = dict(W=np.float64, nasa=np.float64, A=np.float64, b=np.float64, Ea=np.float64, rtype=np.uint8,
               reversible=np.uint8, reac_ptr=np.int32, reac_sp=np.int32, reac_nu=np.int32, prod_ptr=np.int32,
               prod_sp=np.int32, prod_nu=np.int32, eff_ptr=np.int32, eff_sp=np.int32, eff_val=np.float64,
               A0=np.float64, b0=np.float64, Ea0=np.float64, troe=np.float64)


class _OracleMech(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32)] + [(f, C.c_void_p) for f in _MECH_FIELDS]


def build(force: bool = False) -> Path:
    """g++ -O2 (no fast-math) + OpenMP, as BASELINE.md's CPU-baseline plan states."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", str(_LIB), str(_SRC)]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.oracle_arrhenius.restype = C.c_double
        _lib.oracle_arrhenius.argtypes = [C.c_double] * 4
    return _lib


class OracleMechanism:
    """Holds contiguous copies of the mechanism arrays and the C struct that points at them."""

    def __init__(self, n_species: int, n_reactions: int, **arrays):
        self.K, self.I = int(n_species), int(n_reactions)
        self._keep = {}
        self.c = _OracleMech()
        self.c.n_species, self.c.n_reactions = self.K, self.I
        for f in _MECH_FIELDS:
            a = np.ascontiguousarray(arrays[f], dtype=_DTYPES[f])
            if a.size == 0:
                a = np.zeros(1, dtype=_DTYPES[f])
            self._keep[f] = a
            setattr(self.c, f, a.ctypes.data)

    @classmethod
    def from_arrays(cls, n_species, n_reactions, arrays: dict):
        return cls(n_species, n_reactions, **arrays)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def evaluate(mech: OracleMechanism, T, P, Y, Yin=None, tau=None, *, want=("kf", "kr", "q", "wdot"),
             long_double: bool = False, nthreads: int = 0) -> dict:
    """O1..O10 over a batch. Y, Yin: [K][N] species-major. Returns dict of requested outputs:
    kf, kr, q: [I][N]; wdot, F: [K][N]."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    P = np.ascontiguousarray(P, dtype=np.float64)
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    N = T.shape[0]
    assert Y.shape == (mech.K, N)
    if Yin is not None:
        Yin = np.ascontiguousarray(Yin, dtype=np.float64)
        tau = np.ascontiguousarray(tau, dtype=np.float64)
    out = {}
    for name in ("kf", "kr", "q"):
        out[name] = np.empty((mech.I, N)) if name in want else None
    for name in ("wdot", "F"):
        out[name] = np.empty((mech.K, N)) if name in want else None
    rc = lib().oracle_eval(C.byref(mech.c), C.c_int64(N), _p(T), _p(P), _p(Y), _p(Yin), _p(tau), C.c_int64(N),
                           _p(out["kf"]), _p(out["kr"]), _p(out["q"]), C.c_int64(N), _p(out["wdot"]),
                           _p(out["F"]), C.c_int(int(long_double)), C.c_int(nthreads))
    if rc != 0:
        raise RuntimeError(f"oracle_eval failed rc={rc}")
    return {k: v for k, v in out.items() if v is not None}


def evaluate_energy(mech: OracleMechanism, T, P, Y, Tin, Yin, tau, *, long_double: bool = False,
                    nthreads: int = 0) -> dict:
    """Adiabatic PSR residual (energy row NEXT-1 + species rows O10).  Returns F [K][N], FT [N], wdot [K][N]."""
    arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (T, P, Y, Tin, Yin, tau)]
    T, P, Y, Tin, Yin, tau = arrs
    N = T.shape[0]
    assert Y.shape == (mech.K, N) and Yin.shape == (mech.K, N) and Tin.shape == (N,)
    F, wdot, FT = np.empty((mech.K, N)), np.empty((mech.K, N)), np.empty(N)
    rc = lib().oracle_eval_energy(C.byref(mech.c), C.c_int64(N), _p(T), _p(P), _p(Y), _p(Tin), _p(Yin), _p(tau),
                                  C.c_int64(N), _p(F), _p(FT), _p(wdot), C.c_int(int(long_double)), C.c_int(nthreads))
    if rc != 0:
        raise RuntimeError(f"oracle_eval_energy failed rc={rc}")
    return dict(F=F, FT=FT, wdot=wdot)


def jacobian(mech: OracleMechanism, T, P, Y, Yin, tau, *, Tin=None, long_double: bool = False, nthreads: int = 0) -> dict:
    """O11. Returns J [N][K+1][K+1] indexed J[r, col, row] (column-major per reactor), F0, S, H: [N][K+1].
    With Tin [N]: row 0 of the residual is the energy row (NEXT-1) instead of T - T_set."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    P = np.ascontiguousarray(P, dtype=np.float64)
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    Yin = np.ascontiguousarray(Yin, dtype=np.float64)
    tau = np.ascontiguousarray(tau, dtype=np.float64)
    N, n = T.shape[0], mech.K + 1
    J = np.empty((N, n, n))
    F0, S, H = np.empty((N, n)), np.empty((N, n)), np.empty((N, n))
    if Tin is not None:
        Tin = np.ascontiguousarray(Tin, dtype=np.float64)
        rc = lib().oracle_jacobian_energy(C.byref(mech.c), C.c_int64(N), _p(T), _p(P), _p(Y), _p(Tin), _p(Yin), _p(tau),
                                          C.c_int64(N), _p(J), _p(F0), _p(S), _p(H), C.c_int(int(long_double)),
                                          C.c_int(nthreads))
    else:
        rc = lib().oracle_jacobian(C.byref(mech.c), C.c_int64(N), _p(T), _p(P), _p(Y), _p(Yin), _p(tau), C.c_int64(N),
                                   _p(J), _p(F0), _p(S), _p(H), C.c_int(int(long_double)), C.c_int(nthreads))
    if rc != 0:
        raise RuntimeError(f"oracle_jacobian failed rc={rc}")
    return dict(J=J, F0=F0, S=S, H=H)


def roundoff_scale(mech: OracleMechanism, T, P, Y, Yin=None, tau=None, *, nthreads: int = 0) -> dict:
    """Round-off scales (floor terms of the parity criteria): Sw [K][N] = sum_k (nu'+nu'')(|kf prod| + |kr prod|)
    (x |[M]| for three-body), and with Yin, tau also SF [K][N] = |Y - Yin|/tau + (W/rho) Sw (= S of jacobian())."""
    T, P, Y = (np.ascontiguousarray(a, dtype=np.float64) for a in (T, P, Y))
    N = T.shape[0]
    Sw = np.empty((mech.K, N))
    SF = None
    if Yin is not None:
        Yin = np.ascontiguousarray(Yin, dtype=np.float64)
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        SF = np.empty((mech.K, N))
    rc = lib().oracle_roundoff_scale(C.byref(mech.c), C.c_int64(N), _p(T), _p(P), _p(Y), _p(Yin), _p(tau), C.c_int64(N),
                                     _p(Sw), _p(SF), C.c_int(nthreads))
    if rc != 0:
        raise RuntimeError(f"oracle_roundoff_scale failed rc={rc}")
    return dict(Sw=Sw, SF=SF) if SF is not None else dict(Sw=Sw)


def lu_solve(A, b, *, long_double: bool = False):
    """NEXT-2: batched A x = b by Gaussian elimination with partial pivoting.  A: [N][n][n] with A[r, j, i] =
    entry (row i, column j) (column-major per system, the layout of J), b: [N][n].  Returns x [N][n], info [N]."""
    A = np.ascontiguousarray(A, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    N, n = b.shape
    assert A.shape == (N, n, n)
    x = np.full((N, n), np.nan)
    info = np.zeros(N, dtype=np.int32)
    lib().oracle_lu_solve(C.c_int64(N), C.c_int(n), _p(A), _p(b), _p(x), _p(info), C.c_int(int(long_double)))
    return x, info


_DETAIL_COLS = ("kinf", "k0", "Pr", "Fcent", "F", "M", "Kp", "Kc", "kf", "kr", "q")


def ptc_step(J, F, dt, *, long_double: bool = False):
    """NEXT-4: one pseudo-transient (implicit Euler) step (I/dt + J) dx = -F per system.
    J: [N][n][n] with J[r, j, i] = entry (row i, column j); F: [N][n]; dt: [N].  Returns dx [N][n], info [N]."""
    J = np.ascontiguousarray(J, dtype=np.float64)
    F = np.ascontiguousarray(F, dtype=np.float64)
    dt = np.ascontiguousarray(dt, dtype=np.float64)
    N, n = F.shape
    assert J.shape == (N, n, n) and dt.shape == (N,)
    dx = np.empty_like(F)
    info = np.zeros(N, dtype=np.int32)
    lib().oracle_ptc_step(C.c_int64(N), C.c_int(n), _p(J), _p(F), _p(dt), _p(dx), _p(info), C.c_int(int(long_double)))
    return dx, info


def detail(mech: OracleMechanism, T: float, P: float, Y) -> dict:
    """Per-reaction intermediates of one reactor (for the pins)."""
    Y = np.ascontiguousarray(Y, dtype=np.float64).reshape(-1)
    rxn = np.empty((mech.I, 11))
    Cc = np.empty(mech.K)
    rho = C.c_double()
    lib().oracle_detail(C.byref(mech.c), C.c_double(T), C.c_double(P), _p(Y), _p(rxn), _p(Cc), C.byref(rho))
    out = {name: rxn[:, i].copy() for i, name in enumerate(_DETAIL_COLS)}
    out["C"] = Cc
    out["rho"] = rho.value
    return out


def arrhenius(A, b, Ea, T) -> float:
    return float(lib().oracle_arrhenius(A, b, Ea, T))


def nasa7(a, T):
    a = np.ascontiguousarray(a, dtype=np.float64)
    cp, h, s = C.c_double(), C.c_double(), C.c_double()
    lib().oracle_nasa7(_p(a), C.c_double(T), C.byref(cp), C.byref(h), C.byref(s))
    return cp.value, h.value, s.value


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def host_cores() -> int:
    return len(os.sched_getaffinity(0))


class SolveOpts(C.Structure):
    """Constants of the hybrid solver (the paper leaves them to its ref. [5]: the caller's)."""
    _fields_ = [("atol", C.c_double), ("rtol", C.c_double), ("max_iter", C.c_int32), ("max_newton", C.c_int32),
                ("max_ptc", C.c_int32), ("reserved", C.c_int32), ("dt0", C.c_double), ("dt_grow", C.c_double),
                ("dt_shrink", C.c_double), ("y_floor", C.c_double)]


def solve_hybrid(mech: OracleMechanism, T, P, Y, Yin, tau, *, Tin=None, atol=1e-12, rtol=1e-8, max_iter=50,
                 max_newton=10, max_ptc=10, dt0=1e-6, dt_grow=2.0, dt_shrink=0.25, y_floor=1e-9, nthreads: int = 0) -> dict:
    """NEXT-4: hybrid Newton / pseudo-transient solve of the PSR equations, one reactor at a time.
    Returns T [N], Y [K][N] (the solution estimates), status [N] (0 converged, 1 budget exhausted), n_newton, n_ptc."""
    T = np.array(T, dtype=np.float64)
    Y = np.array(Y, dtype=np.float64, order="C")
    P, Yin, tau = (np.ascontiguousarray(a, dtype=np.float64) for a in (P, Yin, tau))
    N = T.shape[0]
    assert Y.shape == (mech.K, N) and Yin.shape == (mech.K, N)
    if Tin is not None:
        Tin = np.ascontiguousarray(Tin, dtype=np.float64)
    o = SolveOpts(atol, rtol, max_iter, max_newton, max_ptc, 0, dt0, dt_grow, dt_shrink, y_floor)
    status, nn, npt = (np.zeros(N, dtype=np.int32) for _ in range(3))
    rc = lib().oracle_solve_hybrid(C.byref(mech.c), C.c_int64(N), _p(T), _p(P), _p(Y), _p(Tin), _p(Yin), _p(tau),
                                   C.c_int64(N), C.byref(o), _p(status), _p(nn), _p(npt), C.c_int(nthreads))
    if rc != 0:
        raise RuntimeError(f"oracle_solve_hybrid failed rc={rc}")
    return dict(T=T, Y=Y, status=status, n_newton=nn, n_ptc=npt)
