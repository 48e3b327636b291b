"""Thin ctypes binding over libpsr_b200.so (include/psr.h).  Argument marshalling only: every step
of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and the
current stream.  There is no CPU fallback: a missing library or device raises."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libpsr_b200.so"

OPT_JAC_UNHOISTED, OPT_FUSED_ONLY, OPT_JAC_GENERIC, OPT_NO_TMEM = 1, 2, 3, 4
PSR_OK, PSR_EINVAL, PSR_EUNSUPPORTED, PSR_ENOMEM, PSR_ECUDA, PSR_EIO = range(6)
_STATUS = {0: "PSR_OK", 1: "PSR_EINVAL", 2: "PSR_EUNSUPPORTED", 3: "PSR_ENOMEM", 4: "PSR_ECUDA", 5: "PSR_EIO"}

EXPORTS = ("psr_mech_load", "psr_mech_free", "psr_eval_kf_kr", "psr_eval_wdot", "psr_eval_residual",
           "psr_eval_residual_energy", "psr_fd_jacobian", "psr_fd_jacobian_energy", "psr_lu_solve", "psr_ptc_solve", "psr_last_error", "psr_mech_info", "psr_mech_set_option", "psr_mech_reserve", "psr_fd_jacobian_noalloc", "psr_check_failures", "psr_solve_hybrid", "psr_solve_hybrid_workspace_bytes", "psr_probe_fp64", "psr_probe_exp_values", "psr_version")

_DESC_ARRAYS = (("W", np.float64), ("nasa", np.float64), ("A", np.float64), ("b", np.float64), ("Ea", np.float64),
                ("rtype", np.uint8), ("reversible", np.uint8), ("reac_ptr", np.int32), ("reac_sp", np.int32),
                ("reac_nu", np.int32), ("prod_ptr", np.int32), ("prod_sp", np.int32), ("prod_nu", np.int32),
                ("eff_ptr", np.int32), ("eff_sp", np.int32), ("eff_val", np.float64), ("A0", np.float64),
                ("b0", np.float64), ("Ea0", np.float64), ("troe", np.float64))


class PsrMechDesc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32)] + [(n, C.c_void_p) for n, _ in _DESC_ARRAYS]


class PsrMechInfo(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_species", "n_reactions", "tile", "warps", "chunk_reactions", "n_chunks",
                                         "smem_bytes", "ctas_per_sm", "n_sm", "n_falloff", "n_third_body", "nnz_nu",
                                         "eval_kernel", "eval_parts", "eval_acc_global", "jac_kernel")]


class PsrSolveOpts(C.Structure):
    """psr_solve_opts: the constants of the hybrid solver (the paper leaves them to its ref. [5])."""
    _fields_ = [("atol", C.c_double), ("rtol", C.c_double), ("max_iter", C.c_int32), ("max_newton", C.c_int32),
                ("max_ptc", C.c_int32), ("reserved", C.c_int32), ("dt0", C.c_double), ("dt_grow", C.c_double),
                ("dt_shrink", C.c_double), ("y_floor", C.c_double)]


class PsrError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


_lib = None


def lib():
    """Load (building first if the sources are newer) the C-ABI library.  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        if _build.needs_build():
            _build.build()
        if not _LIB_PATH.exists():
            raise RuntimeError(f"{_LIB_PATH} is missing: the CUDA extension must be built (python -m paper_2005_11468_b200.build)")
        L = C.CDLL(str(_LIB_PATH))
        vp, i64, dp = C.c_void_p, C.c_int64, C.c_void_p
        L.psr_mech_load.argtypes = [C.POINTER(PsrMechDesc), C.POINTER(vp)]
        L.psr_mech_load.restype = C.c_int
        L.psr_mech_free.argtypes = [vp]
        L.psr_mech_free.restype = None
        L.psr_eval_kf_kr.argtypes = [vp, i64, dp, dp, dp, i64, dp, dp, i64, vp]
        L.psr_eval_kf_kr.restype = C.c_int
        L.psr_eval_wdot.argtypes = [vp, i64, dp, dp, dp, i64, dp, dp, i64, vp]
        L.psr_eval_wdot.restype = C.c_int
        L.psr_eval_residual.argtypes = [vp, i64, dp, dp, dp, dp, dp, i64, dp, dp, vp]
        L.psr_eval_residual.restype = C.c_int
        L.psr_eval_residual_energy.argtypes = [vp, i64, dp, dp, dp, dp, dp, dp, i64, dp, dp, dp, vp]
        L.psr_eval_residual_energy.restype = C.c_int
        L.psr_fd_jacobian_energy.argtypes = [vp, i64, dp, dp, dp, dp, dp, dp, i64, dp, dp, vp]
        L.psr_fd_jacobian_energy.restype = C.c_int
        L.psr_lu_solve.argtypes = [i64, C.c_int32, dp, dp, dp, vp]
        L.psr_lu_solve.restype = C.c_int
        L.psr_ptc_solve.argtypes = [i64, C.c_int32, dp, dp, dp, dp, dp, vp]
        L.psr_ptc_solve.restype = C.c_int
        L.psr_fd_jacobian.argtypes = [vp, i64, dp, dp, dp, dp, dp, i64, dp, dp, vp]
        L.psr_fd_jacobian.restype = C.c_int
        L.psr_fd_jacobian_noalloc.argtypes = [vp, i64, dp, dp, dp, dp, dp, i64, dp, dp, vp]
        L.psr_fd_jacobian_noalloc.restype = C.c_int
        L.psr_last_error.argtypes = []
        L.psr_last_error.restype = C.c_char_p
        L.psr_mech_info.argtypes = [vp, C.POINTER(PsrMechInfo)]
        L.psr_mech_info.restype = C.c_int
        L.psr_solve_hybrid_workspace_bytes.argtypes = [vp, i64]
        L.psr_solve_hybrid_workspace_bytes.restype = C.c_size_t
        L.psr_solve_hybrid.argtypes = [vp, i64, dp, dp, dp, dp, dp, dp, i64, C.POINTER(PsrSolveOpts), vp, C.c_size_t, dp, dp, dp, vp]
        L.psr_solve_hybrid.restype = C.c_int
        L.psr_check_failures.argtypes = [C.c_int32, C.POINTER(C.c_int32)]
        L.psr_check_failures.restype = C.c_int32
        L.psr_mech_reserve.argtypes = [vp, i64]
        L.psr_mech_reserve.restype = C.c_int
        L.psr_mech_set_option.argtypes = [vp, C.c_int32, C.c_int32]
        L.psr_mech_set_option.restype = C.c_int
        L.psr_probe_fp64.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.psr_probe_fp64.restype = C.c_int
        L.psr_probe_exp_values.argtypes = [vp, dp, dp, C.c_int32]
        L.psr_probe_exp_values.restype = C.c_int
        L.psr_version.argtypes = []
        L.psr_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(status: int):
    if status != PSR_OK:
        raise PsrError(status, lib().psr_last_error().decode())


def make_desc(n_species: int, n_reactions: int, arrays: dict):
    """Build a psr_mech_desc from numpy arrays; returns (desc, keepalive list)."""
    desc = PsrMechDesc()
    desc.n_species, desc.n_reactions = int(n_species), int(n_reactions)
    keep = []
    for name, dt in _DESC_ARRAYS:
        a = arrays.get(name)
        if a is None:
            setattr(desc, name, None)
            continue
        a = np.ascontiguousarray(a, dtype=dt)
        if a.size == 0:
            a = np.zeros(1, dtype=dt)
        keep.append(a)
        setattr(desc, name, a.ctypes.data)
    return desc, keep


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ld(Y, N):
    """Leading dimension of a species-major [K][N] tensor (row stride; N for degenerate shapes)."""
    return max(int(Y.stride(0)), int(N)) if (Y.dim() == 2 and Y.shape[0] > 1 and Y.shape[1] > 1) else int(N)


def _like(Y, rows, N, ld):
    """A [rows][N] output that shares Y's leading dimension (the C ABI has ONE ld for Y, Yin, F, wdot)."""
    import torch
    if ld == N:
        return torch.empty((rows, N), dtype=torch.float64, device=Y.device)
    return torch.empty((rows, ld), dtype=torch.float64, device=Y.device)[:, :N]


def _chk_ld(name, t, N, ld):
    if t is not None and _ld(t, N) != ld:
        raise ValueError(f"{name} must share the leading dimension of Y ({ld})")


def _chk_dev(name, t, rows=None, N=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64):
        raise TypeError(f"{name}: expected a CUDA float64 tensor")
    if t.dim() == 2 and t.shape[1] > 1 and t.stride(1) != 1:
        raise ValueError(f"{name}: rows must be contiguous (species-major [K][ld])")


class Mechanism:
    """Device-resident mechanism (psr_mech).  Methods mirror the C ABI one-to-one."""

    def __init__(self, n_species: int, n_reactions: int, arrays: dict):
        desc, keep = make_desc(n_species, n_reactions, arrays)
        h = C.c_void_p()
        _check(lib().psr_mech_load(C.byref(desc), C.byref(h)))
        self._h = h
        self.K, self.I = int(n_species), int(n_reactions)

    @classmethod
    def from_synth(cls, mech):
        return cls(mech.n_species, mech.n_reactions, mech.arrays())

    def close(self):
        if getattr(self, "_h", None):
            lib().psr_mech_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self) -> dict:
        inf = PsrMechInfo()
        _check(lib().psr_mech_info(self._h, C.byref(inf)))
        return {n: getattr(inf, n) for n, _ in PsrMechInfo._fields_}

    def reserve(self, N: int):
        """psr_mech_reserve: size the Jacobian sweep's scratch for batches of up to N reactors (before a capture)."""
        _check(lib().psr_mech_reserve(self._h, int(N)))

    def set_option(self, option: int, value: int):
        """psr_mech_set_option: diagnostic switches (OPT_JAC_UNHOISTED, OPT_FUSED_ONLY)."""
        _check(lib().psr_mech_set_option(self._h, int(option), int(value)))

    def probe_exp_values(self, x):
        """The kernels' exp on a host float64 array (diagnostic, psr_probe_exp_values)."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.empty_like(x)
        _check(lib().psr_probe_exp_values(self._h, x.ctypes.data, y.ctypes.data, x.size))
        return y

    # --- psr_eval_kf_kr
    def eval_kf_kr(self, T, P, Y, kf=None, kr=None):
        import torch
        N = T.shape[0]
        ld = _ld(Y, N)
        for nm, t in (("T", T), ("P", P), ("Y", Y)):
            _chk_dev(nm, t)
        if kf is None:
            kf = torch.empty((self.I, N), dtype=torch.float64, device=T.device)
        if kr is None:
            kr = torch.empty((self.I, N), dtype=torch.float64, device=T.device)
        _check(lib().psr_eval_kf_kr(self._h, N, _ptr(T), _ptr(P), _ptr(Y), ld, _ptr(kf), _ptr(kr), _ld(kf, N), _stream()))
        return kf, kr

    # --- psr_eval_wdot
    def eval_wdot(self, T, P, Y, wdot=None, q=None, want_q=False):
        import torch
        N = T.shape[0]
        ld = _ld(Y, N)
        for nm, t in (("T", T), ("P", P), ("Y", Y)):
            _chk_dev(nm, t)
        if wdot is None:
            wdot = _like(Y, self.K, N, ld)
        if q is None and want_q:
            q = torch.empty((self.I, N), dtype=torch.float64, device=T.device)
        _chk_ld("wdot", wdot, N, ld)
        _check(lib().psr_eval_wdot(self._h, N, _ptr(T), _ptr(P), _ptr(Y), ld, _ptr(wdot), _ptr(q),
                                   _ld(q, N) if q is not None else 0, _stream()))
        return (wdot, q) if (want_q or q is not None) else wdot

    # --- psr_eval_residual
    def eval_residual(self, T, P, Y, Yin, tau, F=None, wdot=None, want_wdot=False):
        import torch
        N = T.shape[0]
        ld = _ld(Y, N)
        for nm, t in (("T", T), ("P", P), ("Y", Y), ("Yin", Yin), ("tau", tau)):
            _chk_dev(nm, t)
        if F is None:
            F = _like(Y, self.K, N, ld)
        if wdot is None and want_wdot:
            wdot = _like(Y, self.K, N, ld)
        for nm, t in (("Yin", Yin), ("F", F), ("wdot", wdot)):
            _chk_ld(nm, t, N, ld)
        _check(lib().psr_eval_residual(self._h, N, _ptr(T), _ptr(P), _ptr(Y), _ptr(Yin), _ptr(tau), ld, _ptr(F),
                                       _ptr(wdot), _stream()))
        return (F, wdot) if wdot is not None else F

    # --- psr_eval_residual_energy
    def eval_residual_energy(self, T, P, Y, Tin, Yin, tau, F=None, FT=None, wdot=None, want_wdot=False):
        import torch
        N = T.shape[0]
        ld = _ld(Y, N)
        for nm, t in (("T", T), ("P", P), ("Y", Y), ("Tin", Tin), ("Yin", Yin), ("tau", tau)):
            _chk_dev(nm, t)
        if F is None:
            F = _like(Y, self.K, N, ld)
        if FT is None:
            FT = torch.empty_like(T)
        if wdot is None and want_wdot:
            wdot = _like(Y, self.K, N, ld)
        for nm, t in (("Yin", Yin), ("F", F), ("wdot", wdot)):
            _chk_ld(nm, t, N, ld)
        _check(lib().psr_eval_residual_energy(self._h, N, _ptr(T), _ptr(P), _ptr(Y), _ptr(Tin), _ptr(Yin), _ptr(tau),
                                              ld, _ptr(F), _ptr(FT), _ptr(wdot), _stream()))
        return (F, FT, wdot) if wdot is not None else (F, FT)

    # --- psr_fd_jacobian
    def fd_jacobian(self, T, P, Y, Yin, tau, J=None, F0=None, want_F0=False, Tin=None):
        """Tin given: psr_fd_jacobian_energy (row 0 = energy row), else psr_fd_jacobian (row 0 = T - T_set)."""
        import torch
        N = T.shape[0]
        ld = _ld(Y, N)
        n = self.K + 1
        for nm, t in (("T", T), ("P", P), ("Y", Y), ("Yin", Yin), ("tau", tau)) + ((("Tin", Tin),) if Tin is not None else ()):
            _chk_dev(nm, t)
        _chk_ld("Yin", Yin, N, ld)
        if J is None:
            J = torch.empty((N, n, n), dtype=torch.float64, device=T.device)  # J[r, col, row]
        if F0 is None and want_F0:
            F0 = torch.empty((N, n), dtype=torch.float64, device=T.device)
        if Tin is not None:
            _check(lib().psr_fd_jacobian_energy(self._h, N, _ptr(T), _ptr(P), _ptr(Y), _ptr(Tin), _ptr(Yin), _ptr(tau),
                                                ld, _ptr(J), _ptr(F0), _stream()))
        else:
            _check(lib().psr_fd_jacobian(self._h, N, _ptr(T), _ptr(P), _ptr(Y), _ptr(Yin), _ptr(tau), ld, _ptr(J),
                                         _ptr(F0), _stream()))
        return (J, F0) if F0 is not None else J


def _solve_hybrid(self, T, P, Y, Yin, tau, Tin=None, workspace=None, atol=1e-12, rtol=1e-8, max_iter=50, max_newton=10,
                  max_ptc=10, dt0=1e-6, dt_grow=2.0, dt_shrink=0.25, y_floor=1e-9):
    """psr_solve_hybrid: T [N] and Y [K][ld] hold the initial estimate and are overwritten by the solution estimate.
    Returns (status, n_newton, n_ptc) int32 [N].  workspace: a CUDA uint8 tensor (allocated for the whole batch if
    None; a smaller one makes the call work through the batch in sub-batches)."""
    import torch
    N = T.shape[0]
    ld = _ld(Y, N)
    for nm, t in (("T", T), ("P", P), ("Y", Y), ("Yin", Yin), ("tau", tau)) + ((("Tin", Tin),) if Tin is not None else ()):
        _chk_dev(nm, t)
    _chk_ld("Yin", Yin, N, ld)
    if workspace is None:
        workspace = torch.empty(int(lib().psr_solve_hybrid_workspace_bytes(self._h, max(N, 1))), dtype=torch.uint8, device=T.device)
    opts = PsrSolveOpts(atol, rtol, max_iter, max_newton, max_ptc, 0, dt0, dt_grow, dt_shrink, y_floor)
    status, nn, npt = (torch.empty(N, dtype=torch.int32, device=T.device) for _ in range(3))
    self.reserve(N)
    _check(lib().psr_solve_hybrid(self._h, N, _ptr(T), _ptr(P), _ptr(Y), _ptr(Tin), _ptr(Yin), _ptr(tau), ld, C.byref(opts),
                                  _ptr(workspace), workspace.numel(), _ptr(status), _ptr(nn), _ptr(npt), _stream()))
    return status, nn, npt


Mechanism.solve_hybrid = _solve_hybrid


def _fd_jacobian_noalloc(self, T, P, Y, Yin, tau, J, F0=None):
    """psr_fd_jacobian_noalloc: the caller passes every array (J [N][n][n], F0 [N][n] or None); the library allocates
    nothing (its scratch is a static device array).  Returns J."""
    N = T.shape[0]
    ld = _ld(Y, N)
    n = self.K + 1
    for nm, t in (("T", T), ("P", P), ("Y", Y), ("Yin", Yin), ("tau", tau), ("J", J)) + ((("F0", F0),) if F0 is not None else ()):
        _chk_dev(nm, t)
    _chk_ld("Yin", Yin, N, ld)
    if tuple(J.shape) != (N, n, n) or not J.is_contiguous() or (F0 is not None and (tuple(F0.shape) != (N, n) or not F0.is_contiguous())):
        raise ValueError("J must be contiguous [N][K+1][K+1] and F0 contiguous [N][K+1]")
    _check(lib().psr_fd_jacobian_noalloc(self._h, N, _ptr(T), _ptr(P), _ptr(Y), _ptr(Yin), _ptr(tau), ld, _ptr(J), _ptr(F0), _stream()))
    return J


Mechanism.fd_jacobian_noalloc = _fd_jacobian_noalloc


def check_failures(selftest: bool = False):
    """psr_check_failures: (count, first_code) of the bounds-checked build; count is -1 in the product build."""
    code = C.c_int32(0)
    n = lib().psr_check_failures(1 if selftest else 0, C.byref(code))
    return int(n), int(code.value)


def probe_fp64(kind: int, iters: int):
    """(elapsed_ms, ops) of the FP64 pipe probe (0 DFMA, 1 exp, 2 log)."""
    ms, ops = C.c_double(), C.c_double()
    _check(lib().psr_probe_fp64(kind, iters, C.byref(ms), C.byref(ops)))
    return ms.value, ops.value


def version() -> str:
    return lib().psr_version().decode()


def lu_solve(A, b, info=None):
    """psr_lu_solve: A [N][n][n] (A[r, col, row], the layout of J), b [N][n] overwritten by the solution.
    Returns (b, info) with info [N] int32 (0 = solved)."""
    import torch
    N, n = b.shape
    if A.shape != (N, n, n) or not A.is_contiguous() or not b.is_contiguous():
        raise ValueError("A must be contiguous [N][n][n] and b contiguous [N][n]")
    for nm, t in (("A", A), ("b", b)):
        _chk_dev(nm, t)
    if info is None:
        info = torch.empty(N, dtype=torch.int32, device=b.device)
    _check(lib().psr_lu_solve(N, n, _ptr(A), _ptr(b), _ptr(info), _stream()))
    return b, info


def ptc_solve(J, F, dt, dx=None, info=None):
    """psr_ptc_solve: one pseudo-transient step (I/dt + J) dx = -F per reactor.  J [N][n][n] (J[r, col, row]),
    F [N][n], dt [N]; returns (dx [N][n], info [N] int32)."""
    import torch
    N, n = F.shape
    if J.shape != (N, n, n) or dt.shape != (N,) or not (J.is_contiguous() and F.is_contiguous() and dt.is_contiguous()):
        raise ValueError("J must be contiguous [N][n][n], F contiguous [N][n], dt contiguous [N]")
    for nm, t in (("J", J), ("F", F), ("dt", dt)):
        _chk_dev(nm, t)
    if dx is None:
        dx = torch.empty_like(F)
    if info is None:
        info = torch.empty(N, dtype=torch.int32, device=F.device)
    _check(lib().psr_ptc_solve(N, n, _ptr(J), _ptr(F), _ptr(dt), _ptr(dx), _ptr(info), _stream()))
    return dx, info
