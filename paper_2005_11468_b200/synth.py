"""Seeded synthetic mechanisms and reactor states (BASELINE.json: configs C0..C4).

This module builds INPUTS only: species, NASA-7 coefficients, reaction lists, rate
parameters and reactor states, all as numpy arrays.  It contains none of the method's
arithmetic (no rate constants, no thermo evaluation, no residual) and is the one module
that both the CUDA path (tests, bench.py) and the oracle tests draw inputs from.

The synthetic mechanisms stand in for the real ones the paper measures on (GRI-size
53/325; Appel et al. 101/542), which are not reconstructed here.

Recipe (SURVEY.md section 8(c) readings g7-g12, 8(d)):
  species   : random (C,H,O,N) atom vectors, C,N in 0..2, H in 0..4, O in 0..2, non-zero;
              a share of species are sums of two earlier ones (so balanced reactions exist
              even at K=10); W from atomic masses C 12.011, H 1.008, O 15.999, N 14.007.
  thermo    : a0~U(2.5,4.5), a1~U(+-1e-3), a2~U(+-1e-6), a3~U(+-1e-10), a4~U(+-1e-14),
              a5~U(+-3e4), a6~U(-5,15); single temperature range.
  reactions : m in 1..mmax species per side drawn with replacement (nu in 1..3), no species
              on both sides, element balanced (bucket multisets by element vector and pair
              them); A log-uniform 1e6..1e14, b~U(-2,2), Ea~U(0,50) kcal/mol (stored cal/mol).
  3rd body  : n_tb reactions get efficiency lists of 2..min(6,K) distinct species, alpha~U(.5,5).
  Troe      : n_troe other reactions; alpha~U(.3,.9), T***~U(50,500), T*~U(500,3000),
              T**~U(3000,8000); low-pressure b0, Ea0 from the same laws, log10 A0 =
              log10 A + U(4,7) so that P_r straddles 1; unit efficiencies.
  states    : T~U, P const or log-uniform (atm -> dyn/cm^2), Y~Dirichlet(alpha) floored at
              1e-20 and renormalised; tau log-U(1e-4,1e-2) s; Y_in ~ Dirichlet(1).
Seeds: mechanism 1000+c, state 2000+c for config c.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from itertools import combinations_with_replacement

import numpy as np

ATOMIC_MASS = np.array([12.011, 1.008, 15.999, 14.007])  # C, H, O, N
ATOM_MAX = np.array([2, 4, 2, 2])
P_ATM_CGS = 1.01325e6  # dyn/cm^2 per atm (unit conversion of an input, not method arithmetic)

RTYPE_PLAIN, RTYPE_THREE_BODY, RTYPE_LINDEMANN, RTYPE_TROE = 0, 1, 2, 3


@dataclass
class Mechanism:
    """Host-side mechanism description; field names follow include/psr.h: psr_mech_desc."""
    n_species: int
    n_reactions: int
    atoms: np.ndarray       # [K][4] int32 (C,H,O,N) - generator bookkeeping, not passed to the library
    W: np.ndarray           # [K]
    nasa: np.ndarray        # [K][7]
    A: np.ndarray
    b: np.ndarray
    Ea: np.ndarray          # cal/mol
    rtype: np.ndarray       # uint8
    reversible: np.ndarray  # uint8
    reac_ptr: np.ndarray
    reac_sp: np.ndarray
    reac_nu: np.ndarray
    prod_ptr: np.ndarray
    prod_sp: np.ndarray
    prod_nu: np.ndarray
    eff_ptr: np.ndarray
    eff_sp: np.ndarray
    eff_val: np.ndarray
    A0: np.ndarray
    b0: np.ndarray
    Ea0: np.ndarray
    troe: np.ndarray        # [I][4] alpha, T3, T1, T2
    meta: dict = field(default_factory=dict)

    def arrays(self) -> dict:
        return {k: getattr(self, k) for k in (
            "W", "nasa", "A", "b", "Ea", "rtype", "reversible", "reac_ptr", "reac_sp", "reac_nu",
            "prod_ptr", "prod_sp", "prod_nu", "eff_ptr", "eff_sp", "eff_val", "A0", "b0", "Ea0", "troe")}


@dataclass
class ReactorBatch:
    """Species-major SoA state: Y[k, r] is species k of reactor r (include/psr.h layout)."""
    T: np.ndarray    # [N] K
    P: np.ndarray    # [N] dyn/cm^2
    Y: np.ndarray    # [K][N]
    Yin: np.ndarray  # [K][N]
    tau: np.ndarray  # [N] s

    @property
    def n(self) -> int:
        return int(self.T.shape[0])

    def take(self, idx) -> "ReactorBatch":
        idx = np.asarray(idx)
        return ReactorBatch(self.T[idx].copy(), self.P[idx].copy(), np.ascontiguousarray(self.Y[:, idx]),
                            np.ascontiguousarray(self.Yin[:, idx]), self.tau[idx].copy())


# ----------------------------------------------------------------------------- species
def _draw_species_atoms(rng: np.random.Generator, K: int) -> np.ndarray:
    """About half random small atom vectors, the rest sums of two earlier species (bounded
    retries) so that element-balanced reactions exist even for K=10 (SURVEY.md 8(d) pitfall).
    Repeated atom vectors (isomers) are allowed; with 134 possible vectors they are
    unavoidable at K>=200."""
    atoms = np.zeros((K, 4), dtype=np.int32)
    n_base = max(3, (K + 1) // 2)
    for k in range(K):
        made = False
        if k >= n_base:
            for _ in range(64):
                i, j = rng.integers(0, k, size=2)
                s = atoms[i] + atoms[j]
                if np.all(s <= ATOM_MAX):
                    atoms[k] = s
                    made = True
                    break
        if not made:
            while True:
                # small counts: keep sums of two inside the bounds often enough
                v = np.array([rng.integers(0, 2), rng.integers(0, 3), rng.integers(0, 2), rng.integers(0, 2)])
                if k >= n_base:  # fallback draw over the full range
                    v = np.array([rng.integers(0, ATOM_MAX[a] + 1) for a in range(4)])
                if v.sum() > 0:
                    atoms[k] = v
                    break
    return atoms


# ----------------------------------------------------------------------------- reactions
def _multiset_pool(rng: np.random.Generator, K: int, mmax: int, max_triples: int = 400_000) -> np.ndarray:
    """All multisets of 1..min(mmax,2) species, plus all (or a random sample of) triples, as an
    [n][3] int32 array of sorted species indices padded with -1."""
    rows = [np.stack([np.arange(K), np.full(K, -1), np.full(K, -1)], axis=1)]
    if mmax >= 2:
        i, j = np.triu_indices(K)
        rows.append(np.stack([i, j, np.full(i.size, -1)], axis=1))
    if mmax >= 3:
        n_tri = K * (K + 1) * (K + 2) // 6
        if n_tri <= max_triples:
            tri = np.array(list(combinations_with_replacement(range(K), 3)), dtype=np.int64)
        else:
            tri = np.unique(np.sort(rng.integers(0, K, size=(max_triples, 3)), axis=1), axis=0)
        rows.append(tri)
    return np.concatenate(rows, axis=0).astype(np.int32)


def _draw_reactions(rng: np.random.Generator, atoms: np.ndarray, I: int, mmax: int):
    """Ordered (reactants, products) pairs of multisets with equal element sums and disjoint
    species.  If fewer than I distinct pairs exist, stoichiometries repeat (a CHEMKIN
    'duplicate' reaction with fresh rate parameters)."""
    K = atoms.shape[0]
    pool = _multiset_pool(rng, K, mmax)
    padded = np.vstack([atoms, np.zeros((1, 4), dtype=atoms.dtype)])       # index -1 -> zero atoms
    esum = padded[pool].sum(axis=1)                                         # [n][4]
    key = ((esum[:, 0] * 32 + esum[:, 1]) * 32 + esum[:, 2]) * 32 + esum[:, 3]
    order = np.argsort(key, kind="stable")
    pool, key = pool[order], key[order]
    _, b_start, b_len = np.unique(key, return_index=True, return_counts=True)
    bucket_of = np.repeat(np.arange(b_start.size), b_len)
    size_of = (pool >= 0).sum(axis=1)
    elig = b_len[bucket_of] >= 2
    eligible_by_size = [np.nonzero(elig & (size_of == m))[0] for m in range(1, mmax + 1)]
    sizes = [m for m in range(mmax) if eligible_by_size[m].size]
    if not sizes:
        raise RuntimeError("no element-balanced reaction exists for this species set")
    seen: set = set()
    out = []
    tries = 0
    allow_dup = False
    while len(out) < I:
        tries += 1
        if tries > 200 * I and not allow_dup:
            allow_dup = True  # pool exhausted: permit duplicates
        if tries > 2000 * I:
            raise RuntimeError("reaction sampler did not terminate")
        eligible = eligible_by_size[sizes[int(rng.integers(0, len(sizes)))]]   # reactant count uniform in 1..mmax (g10)
        ia = int(eligible[rng.integers(0, eligible.size)])
        bk = bucket_of[ia]
        ib = int(b_start[bk] + rng.integers(0, b_len[bk]))
        if ib == ia:
            continue
        ra = tuple(int(x) for x in pool[ia] if x >= 0)
        rb = tuple(int(x) for x in pool[ib] if x >= 0)
        if set(ra) & set(rb):
            continue
        if (ra, rb) in seen and not allow_dup:
            continue
        seen.add((ra, rb))
        out.append((ra, rb))
    return out


def _side_csr(sides):
    ptr = [0]
    sp, nu = [], []
    for ms in sides:
        uniq = sorted(set(ms))
        for s in uniq:
            sp.append(s)
            nu.append(ms.count(s))
        ptr.append(len(sp))
    return (np.asarray(ptr, dtype=np.int32), np.asarray(sp, dtype=np.int32), np.asarray(nu, dtype=np.int32))


def make_mechanism(n_species: int, n_reactions: int, n_third_body: int, n_troe: int, seed: int,
                   mmax: int = 3, n_lindemann: int = 0) -> Mechanism:
    rng = np.random.default_rng(np.random.PCG64(seed))
    K, I = n_species, n_reactions
    atoms = _draw_species_atoms(rng, K)
    W = atoms.astype(np.float64) @ ATOMIC_MASS
    lo = np.array([2.5, -1e-3, -1e-6, -1e-10, -1e-14, -3e4, -5.0])
    hi = np.array([4.5, 1e-3, 1e-6, 1e-10, 1e-14, 3e4, 15.0])
    nasa = rng.uniform(lo, hi, size=(K, 7))

    rx = _draw_reactions(rng, atoms, I, mmax)
    reac_ptr, reac_sp, reac_nu = _side_csr([r for r, _ in rx])
    prod_ptr, prod_sp, prod_nu = _side_csr([p for _, p in rx])

    A = 10.0 ** rng.uniform(6.0, 14.0, size=I)
    b = rng.uniform(-2.0, 2.0, size=I)
    Ea = rng.uniform(0.0, 50.0, size=I) * 1000.0  # kcal/mol -> cal/mol

    # disjoint third-body / falloff sets (SURVEY reading g7)
    perm = rng.permutation(I)
    tb_idx = np.sort(perm[:n_third_body])
    troe_idx = np.sort(perm[n_third_body:n_third_body + n_troe])
    lind_idx = np.sort(perm[n_third_body + n_troe:n_third_body + n_troe + n_lindemann])
    rtype = np.zeros(I, dtype=np.uint8)
    rtype[tb_idx] = RTYPE_THREE_BODY
    rtype[troe_idx] = RTYPE_TROE
    rtype[lind_idx] = RTYPE_LINDEMANN
    reversible = np.ones(I, dtype=np.uint8)

    eff_ptr = np.zeros(I + 1, dtype=np.int32)
    eff_sp, eff_val = [], []
    tb_set = set(int(x) for x in tb_idx)
    for k in range(I):
        if k in tb_set:
            n_eff = int(rng.integers(2, min(6, K) + 1))
            sp = np.sort(rng.choice(K, size=n_eff, replace=False))
            eff_sp += [int(s) for s in sp]
            eff_val += [float(v) for v in rng.uniform(0.5, 5.0, size=n_eff)]
        eff_ptr[k + 1] = len(eff_sp)

    A0 = np.zeros(I)
    b0 = np.zeros(I)
    Ea0 = np.zeros(I)
    troe = np.zeros((I, 4))
    fall = np.sort(np.concatenate([troe_idx, lind_idx])).astype(np.int64)
    if fall.size:
        A0[fall] = A[fall] * 10.0 ** rng.uniform(4.0, 7.0, size=fall.size)
        b0[fall] = rng.uniform(-2.0, 2.0, size=fall.size)
        Ea0[fall] = rng.uniform(0.0, 50.0, size=fall.size) * 1000.0
    if troe_idx.size:
        n = troe_idx.size
        troe[troe_idx, 0] = rng.uniform(0.3, 0.9, size=n)
        troe[troe_idx, 1] = rng.uniform(50.0, 500.0, size=n)
        troe[troe_idx, 2] = rng.uniform(500.0, 3000.0, size=n)
        troe[troe_idx, 3] = rng.uniform(3000.0, 8000.0, size=n)

    return Mechanism(
        n_species=K, n_reactions=I, atoms=atoms, W=W, nasa=np.ascontiguousarray(nasa),
        A=A, b=b, Ea=Ea, rtype=rtype, reversible=reversible,
        reac_ptr=reac_ptr, reac_sp=reac_sp, reac_nu=reac_nu,
        prod_ptr=prod_ptr, prod_sp=prod_sp, prod_nu=prod_nu,
        eff_ptr=eff_ptr, eff_sp=np.asarray(eff_sp, dtype=np.int32), eff_val=np.asarray(eff_val, dtype=np.float64),
        A0=A0, b0=b0, Ea0=Ea0, troe=np.ascontiguousarray(troe),
        meta={"seed": seed, "n_third_body": n_third_body, "n_troe": n_troe, "n_lindemann": n_lindemann, "mmax": mmax})


# ----------------------------------------------------------------------------- states
def _dirichlet_floored(rng, alpha: float, K: int, N: int) -> np.ndarray:
    y = rng.dirichlet(np.full(K, alpha), size=N)        # [N][K]
    y = np.maximum(y, 1e-20)
    y /= y.sum(axis=1, keepdims=True)                    # reading g11
    return np.ascontiguousarray(y.T)                     # species-major [K][N]


def make_states(K: int, N: int, seed: int, T_range=(800.0, 2500.0), P_atm=(1.0, 1.0),
                dirichlet_alpha: float = 1.0) -> ReactorBatch:
    rng = np.random.default_rng(np.random.PCG64(seed))
    T = rng.uniform(T_range[0], T_range[1], size=N)
    if P_atm[0] == P_atm[1]:
        P = np.full(N, P_atm[0] * P_ATM_CGS)
    else:
        P = np.exp(rng.uniform(np.log(P_atm[0]), np.log(P_atm[1]), size=N)) * P_ATM_CGS
    Y = _dirichlet_floored(rng, dirichlet_alpha, K, N)
    tau = np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), size=N))
    Yin = _dirichlet_floored(rng, 1.0, K, N)
    return ReactorBatch(T=T, P=P, Y=Y, Yin=Yin, tau=tau)


def make_uniform_states(mech: "Mechanism", N: int, seed: int, T: float = 1800.0, P_atm: float = 1.0, tau: float = 50e-3,
                        inlet_X=(0.15, 0.18, 0.67)) -> ReactorBatch:
    """The shape of the paper's timing experiment: N identical reactors at T = 1800 K,
    tau = 50 ms, 1 atm, inlet mole fractions 0.15 / 0.18 / 0.67 on three species (stand-ins for the
    fuel, oxidiser and diluent of a mechanism that is not in this container: species 0, 1, 2).  The reactor
    composition is the same for every reactor: half the inlet, half one seeded Dirichlet(1) draw, so that
    every reaction has non-zero rates."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    K = mech.n_species
    x = np.zeros(K)
    x[:3] = inlet_X
    yin = x * mech.W
    yin /= yin.sum()
    y = 0.5 * yin + 0.5 * _dirichlet_floored(rng, 1.0, K, 1)[:, 0]
    y /= y.sum()
    rep = lambda v: np.ascontiguousarray(np.repeat(v[:, None], N, axis=1))
    return ReactorBatch(T=np.full(N, T), P=np.full(N, P_atm * P_ATM_CGS), Y=rep(y), Yin=rep(yin), tau=np.full(N, tau))


# ----------------------------------------------------------------------------- configs
CONFIGS = {
    # name: mechanism kwargs, state kwargs, N  (BASELINE.json: configs, zero-indexed)
    "C0": dict(mech=dict(n_species=10, n_reactions=20, n_third_body=2, n_troe=0, mmax=2), mech_cfg=0,
               state=dict(T_range=(800.0, 2500.0), P_atm=(1.0, 1.0), dirichlet_alpha=1.0), N=1024),
    "C1": dict(mech=dict(n_species=53, n_reactions=325, n_third_body=28, n_troe=29, mmax=3), mech_cfg=1,
               state=dict(T_range=(800.0, 2500.0), P_atm=(0.5, 10.0), dirichlet_alpha=1.0), N=65536),
    "C2": dict(mech=dict(n_species=200, n_reactions=1500, n_third_body=120, n_troe=100, mmax=3), mech_cfg=2,
               state=dict(T_range=(1000.0, 2200.0), P_atm=(1.0, 1.0), dirichlet_alpha=0.5), N=32768),
    "C3": dict(mech=dict(n_species=500, n_reactions=2500, n_third_body=200, n_troe=150, mmax=3), mech_cfg=3,
               state=dict(T_range=(800.0, 2500.0), P_atm=(1.0, 20.0), dirichlet_alpha=1.0), N=16384),
    # C4: the C1 mechanism (same mechanism seed), its own state seed
    "C4": dict(mech=dict(n_species=53, n_reactions=325, n_third_body=28, n_troe=29, mmax=3), mech_cfg=1,
               state=dict(T_range=(800.0, 2500.0), P_atm=(0.5, 10.0), dirichlet_alpha=1.0), N=8192),
    # P5: the SHAPE of the paper's speed-up experiment, 101 species / 542 reactions
    # (PAPER.md:137), identical reactors at 1800 K, 50 ms (make_uniform_states); batch swept by bench.py --sweep
    "P5": dict(mech=dict(n_species=101, n_reactions=542, n_third_body=47, n_troe=48, mmax=3), mech_cfg=5,
               state=None, N=10000),
}


def make_config(name: str, n_reactors: int | None = None):
    """Return (Mechanism, ReactorBatch) for config 'C0'..'C4' (BASELINE.json) or 'P5' (paper-shaped sweep). n_reactors overrides the batch size
    (the state stream is seeded per config, so the first n reactors of a larger draw differ from a
    smaller draw; parity tests always pass the same arrays to both sides)."""
    cfg = CONFIGS[name]
    c = int(name[1:])
    mech = make_mechanism(seed=1000 + cfg["mech_cfg"], **cfg["mech"])
    N = cfg["N"] if n_reactors is None else int(n_reactors)
    if cfg["state"] is None:
        return mech, make_uniform_states(mech, N, seed=2000 + c)
    batch = make_states(mech.n_species, N, seed=2000 + c, **cfg["state"])
    return mech, batch


def toy_t3():
    """The 3-species toy mechanism T3 of SURVEY.md section 8(c): S0+S1<=>S2 (plain),
    S2+M<=>S0+S1+M (three-body), S0+S1(+M)<=>S2 (Troe).  Inputs only."""
    W = np.array([2.016, 31.998, 34.014])
    nasa = np.array([[3.5, 1e-4, 0.0, 0.0, 0.0, -1000.0, -3.0],
                     [3.7, 2e-4, -1e-8, 0.0, 0.0, -1200.0, 3.5],
                     [4.2, 5e-4, -5e-8, 1e-12, 0.0, -17000.0, 4.0]])
    rx = [((0, 1), (2,)), ((2,), (0, 1)), ((0, 1), (2,))]
    reac_ptr, reac_sp, reac_nu = _side_csr([r for r, _ in rx])
    prod_ptr, prod_sp, prod_nu = _side_csr([p for _, p in rx])
    mech = Mechanism(
        n_species=3, n_reactions=3, atoms=np.zeros((3, 4), dtype=np.int32), W=W, nasa=nasa,
        A=np.array([1e8, 5e11, 2e9]), b=np.array([0.0, -0.5, 0.2]), Ea=np.array([10e3, 45e3, 5e3]),
        rtype=np.array([0, 1, 3], dtype=np.uint8), reversible=np.ones(3, dtype=np.uint8),
        reac_ptr=reac_ptr, reac_sp=reac_sp, reac_nu=reac_nu,
        prod_ptr=prod_ptr, prod_sp=prod_sp, prod_nu=prod_nu,
        eff_ptr=np.array([0, 0, 2, 2], dtype=np.int32), eff_sp=np.array([0, 2], dtype=np.int32),
        eff_val=np.array([2.5, 0.7]),
        A0=np.array([0.0, 0.0, 4e17]), b0=np.array([0.0, 0.0, -1.0]), Ea0=np.array([0.0, 0.0, 3e3]),
        troe=np.array([[0, 0, 0, 0], [0, 0, 0, 0], [0.6, 200.0, 1500.0, 5000.0]], dtype=np.float64),
        meta={"name": "T3"})
    batch = ReactorBatch(T=np.array([1500.0]), P=np.array([P_ATM_CGS]),
                         Y=np.array([[0.1], [0.895], [0.005]]), Yin=np.array([[0.2], [0.8], [0.0]]),
                         tau=np.array([1e-3]))
    return mech, batch
