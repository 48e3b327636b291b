"""Helpers shared by the tests: marshal synth inputs into the oracle, parity metrics (DESIGN.md
'Tolerances', SURVEY.md reading g16)."""
import numpy as np

from oracle import oracle as orc


def oracle_mech(mech):
    return orc.OracleMechanism.from_arrays(mech.n_species, mech.n_reactions, mech.arrays())


def rel_err(a, b):
    """Plain element-wise relative error |a-b|/|b| (b nonzero), 0 where both are exactly equal."""
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    d = np.abs(a - b)
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(d == 0, 0.0, d / np.abs(b))
    return r


def wdot_masked_rel_err(w, w_ref):
    """BASELINE.json: north_star: relative error wherever |wdot| > 1e-12 max|wdot|, the max taken
    over the species of the same reactor (reading g16).  w: [K][N]."""
    w, w_ref = np.asarray(w), np.asarray(w_ref)
    scale = np.abs(w_ref).max(axis=0, keepdims=True)
    mask = np.abs(w_ref) > 1e-12 * scale
    r = rel_err(w, w_ref)
    return np.where(mask, r, 0.0), mask


def residual_rel_err(F, F_ref):
    """Reading g16: relative to max(|F_i|, 1e-12 max_i |F_i|) per reactor. F: [K][N]."""
    F, F_ref = np.asarray(F), np.asarray(F_ref)
    scale = np.abs(F_ref).max(axis=0, keepdims=True)
    den = np.maximum(np.abs(F_ref), 1e-12 * scale)
    den = np.where(den == 0, 1.0, den)
    return np.abs(F - F_ref) / den


EPS = 2.0 ** -53


def jacobian_floor_ratio(J, J_star, S, H, K_y=32.0, K_T=1024.0):
    """SURVEY.md 8(c)-J criterion (1): |J - J*|_ij <= 1e-9 |J*_ij| + K_j eps S_i / h_j.
    J, J_star: [N][col][row]; S, H: [N][n].  Returns the worst ratio lhs / rhs (<=1 passes) and
    the worst 'floor ratio' |J-J*| / (eps S_i / h_j) per column class (T, Y)."""
    J, J_star = np.asarray(J), np.asarray(J_star)
    N, n, _ = J.shape
    Kj = np.full(n, K_y)
    Kj[0] = K_T
    floor = EPS * S[:, None, :] / H[:, :, None]                 # [N][col][row]
    bound = 1e-9 * np.abs(J_star) + Kj[None, :, None] * floor
    diff = np.abs(J - J_star)
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(diff == 0, 0.0, diff / bound)
        fr = np.where(floor > 0, diff / floor, 0.0)
    return float(np.nanmax(ratio)), float(np.nanmax(fr[:, 0, :])), float(np.nanmax(fr[:, 1:, :]))


def floor_criterion(x, x_star, S, K=1024.0, rtol=1e-10, mask=None):
    """Conditioning-aware parity (reading g16b): |x - x*| <= rtol |x*| + K eps S, with x* the
    long-double oracle and S the round-off scale of the entry (oracle.roundoff_scale: the magnitude of the terms
    whose signed sum the entry is).  Where an entry is not the result of cancellation (S ~ |x*|) this is the
    literal relative bound; where it is, no FP64 evaluation -- the oracle included -- can do better than a
    multiple of eps S, the multiple set by the conditioning of the exp arguments (|dG/RT| up to a few hundred),
    hence the same K = 1024 as the T column of the Jacobian criterion.
    Returns (worst lhs/rhs, worst |x - x*| / (eps S))."""
    x, x_star, S = (np.asarray(a, dtype=np.float64) for a in (x, x_star, S))
    diff = np.abs(x - x_star)
    bound = rtol * np.abs(x_star) + K * EPS * S
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(diff == 0, 0.0, diff / bound)
        fr = np.where(S > 0, diff / (EPS * S), 0.0)
    if mask is not None:
        ratio, fr = np.where(mask, ratio, 0.0), np.where(mask, fr, 0.0)
    return float(np.nanmax(ratio)), float(np.nanmax(fr))
