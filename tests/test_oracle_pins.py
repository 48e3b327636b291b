"""Pins for the CPU oracle (oracle/psr_oracle.cpp) -- none of the expected values below comes
from the oracle itself or from the CUDA path.

Sources of truth: (a) tests/golden/t3_pins.json -- the 17-digit values SURVEY.md 8(c) prints for
the toy mechanism T3, which this file first re-derives with mpmath (tests/mp_dense.py: dense
stoichiometric matrices, mp.power, 50 digits); (b) closed forms and invariants that the
equations PAPER.md Eq. 2, 4-9 fix.  Each test names the oracle step (O1..O11) it pins.
"""
import copy
import json
from pathlib import Path

import numpy as np
import pytest
from mpmath import mpf

import mp_dense
from oracle import oracle as orc
from paper_2005_11468_b200 import synth
from util import EPS, jacobian_floor_ratio, oracle_mech, rel_err

GOLD = json.loads((Path(__file__).parent / "golden" / "t3_pins.json").read_text())
RGAS = 8.31446261815324e7
PATM = 1.01325e6


def close(a, b, rtol):
    return abs(float(a) - float(b)) <= rtol * abs(float(b))


@pytest.fixture(scope="module")
def t3():
    mech, batch = synth.toy_t3()
    return mech, batch, oracle_mech(mech)


@pytest.fixture(scope="module")
def t3_mp(t3):
    mech, batch, _ = t3
    return mp_dense.evaluate(mech, batch.T[0], batch.P[0], batch.Y[:, 0], batch.Yin[:, 0], batch.tau[0])


# ------------------------------------------------------------------ the goldens themselves
def test_golden_values_rederived_with_mpmath(t3, t3_mp):
    """The printed T3 values agree with an independent 50-digit dense evaluation to 1e-15."""
    g, m = GOLD, t3_mp
    assert close(m["Wbar"], g["state"]["Wbar"], 1e-15) and close(m["rho"], g["state"]["rho"], 1e-15)
    for i in range(3):
        assert close(m["C"][i], g["state"]["C"][i], 1e-15)
    assert close(m["Ctot"], g["state"]["Ctot"], 1e-15)
    for name, k in (("R0", 0), ("R1", 1), ("R2", 2)):
        for key, val in g[name].items():
            if key in m["rx"][k]:
                assert close(m["rx"][k][key], val, 2e-15), (name, key)
    for i in range(3):
        assert close(m["wdot"][i], g["wdot_sign"][i] * g["wdot_abs"], 2e-15)
    for i in range(1, 4):
        assert close(m["F"][i], g["F"][i], 1e-13)  # F printed with 15-17 digits
    assert m["F"][0] == 0


def test_golden_jacobian_rederived_with_mpmath(t3):
    """Exact difference quotients with the double-precision step h_j = fl(fl(x_j+d_j)-x_j) (g15)."""
    mech, batch, _ = t3
    x = np.concatenate([batch.T, batch.Y[:, 0]])
    base = mp_dense.evaluate(mech, x[0], batch.P[0], x[1:], batch.Yin[:, 0], batch.tau[0], Tset=x[0])
    for j, name in enumerate(("T", "Y0", "Y1", "Y2")):
        delta = 1e-8 * max(abs(x[j]), 1e-10)
        xp = x.copy()
        xp[j] = x[j] + delta
        h = xp[j] - x[j]
        pert = mp_dense.evaluate(mech, xp[0], batch.P[0], xp[1:], batch.Yin[:, 0], batch.tau[0], Tset=x[0])
        col = [(pert["F"][i] - base["F"][i]) / mpf(float(h)) for i in range(4)]
        for i in range(4):
            ref = GOLD["J_cols"][name][i]
            assert abs(float(col[i]) - ref) <= 2e-11 * max(abs(ref), 1e-300) + (0 if ref else 1e-300), (name, i)


def test_g15_step_is_not_delta():
    """For T=1500 the representable step differs from delta by ~5e-9 relative."""
    delta = 1e-8 * 1500.0
    h = (1500.0 + delta) - 1500.0
    assert h == float.fromhex("0x1.f751050000000p-17")
    assert abs(h / delta - 1) > 1e-9


# ------------------------------------------------------------------ O3, O2: closed forms
def test_O3_arrhenius_hand_values():
    for row in GOLD["arrhenius"]:
        got = orc.arrhenius(row["A"], row["b"], row["Ea_kcal"] * 1000.0, row["T"])
        assert close(got, row["k"], 5e-15), row


def test_O3_arrhenius_special_cases():
    # b=0, Ea=0 -> A exactly; Ea=0 -> A T^b; doubling Ea squares the exponential factor
    assert orc.arrhenius(3.0e7, 0.0, 0.0, 1234.5) == 3.0e7
    assert close(orc.arrhenius(2.0, 2.0, 0.0, 1000.0), 2.0e6, 1e-15)
    e1 = orc.arrhenius(1.0, 0.0, 10e3, 1000.0)
    e2 = orc.arrhenius(1.0, 0.0, 20e3, 1000.0)
    assert close(e2, e1 * e1, 1e-14)
    # exp(-Ea/(Rc T)) with Rc = 8.31446261815324/4.184 cal/mol/K
    import math
    assert close(e1, math.exp(-10e3 / (8.31446261815324 / 4.184 * 1000.0)), 1e-15)


def test_O2_nasa_closed_form():
    mech, _ = synth.toy_t3()
    for i, name in enumerate(("S0", "S1", "S2")):
        cp, h, s = orc.nasa7(mech.nasa[i], 1500.0)
        g = GOLD["nasa_T1500"][name]
        assert close(cp, g["cp_R"], 1e-15) and close(h, g["h_RT"], 1e-15) and close(s, g["s_R"], 1e-15)


def test_O2_nasa_thermodynamic_identities():
    """d(h/RT * T)/dT = cp/R and d(s/R)/dT = cp/(R T): central differences on a random species."""
    rng = np.random.default_rng(7)
    a = rng.uniform([2.5, -1e-3, -1e-6, -1e-10, -1e-14, -3e4, -5], [4.5, 1e-3, 1e-6, 1e-10, 1e-14, 3e4, 15])
    T, d = 1300.0, 1e-2
    cp, h, s = orc.nasa7(a, T)
    _, hp, sp = orc.nasa7(a, T + d)
    _, hm, sm = orc.nasa7(a, T - d)
    assert close((hp * (T + d) - hm * (T - d)) / (2 * d), cp, 1e-8)
    assert close((sp - sm) / (2 * d), cp / T, 1e-8)


# ------------------------------------------------------------------ O1, O4-O10 on T3
def test_O1_state_and_ideal_gas_identity(t3):
    mech, batch, om = t3
    d = orc.detail(om, batch.T[0], batch.P[0], batch.Y[:, 0])
    assert close(d["rho"], GOLD["state"]["rho"], 1e-15)
    for i in range(3):
        assert close(d["C"][i], GOLD["state"]["C"][i], 2e-15)
    # identity: sum_i C_i = P/(R T) when C = rho Y/W and rho = P Wbar/(R T)
    assert close(d["C"].sum(), batch.P[0] / (RGAS * batch.T[0]), 1e-15)
    assert close(d["C"].sum(), GOLD["state"]["Ctot"], 1e-15)


def test_O3_to_O8_T3_reactions(t3):
    mech, batch, om = t3
    d = orc.detail(om, batch.T[0], batch.P[0], batch.Y[:, 0])
    for name, k in (("R0", 0), ("R1", 1), ("R2", 2)):
        for key, val in GOLD[name].items():
            if key in d:
                assert close(d[key][k], val, 2e-14), (name, key, d[key][k], val)


def test_O6_lindemann_variant_and_troe_M_scaling(t3):
    mech, batch, om = t3
    lind = copy.deepcopy(mech)
    lind.rtype = np.array([0, 1, 2], dtype=np.uint8)
    d = orc.detail(oracle_mech(lind), batch.T[0], batch.P[0], batch.Y[:, 0])
    assert close(d["kf"][2], GOLD["R2"]["kf_lindemann"], 2e-14)
    # Troe F with [M] scaled by 1e-8 / 1e8: scale A0 instead (P_r = k0 [M] / k_inf is linear in both)
    for scale, key in ((1e-8, "F_M_times_1e-8"), (1e8, "F_M_times_1e8")):
        mm = copy.deepcopy(mech)
        mm.A0 = mech.A0 * scale
        d = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])
        assert close(d["F"][2], GOLD["R2"][key], 5e-14)


def test_O9_O10_T3_wdot_and_residual(t3):
    mech, batch, om = t3
    out = orc.evaluate(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("wdot", "F"))
    for i in range(3):
        assert close(out["wdot"][i, 0], GOLD["wdot_sign"][i] * GOLD["wdot_abs"], 5e-14)
        assert close(out["F"][i, 0], GOLD["F"][i + 1], 5e-14)


# ------------------------------------------------------------------ invariants
def _swap(mech):
    """Swap reactants and products of every reaction (inputs only)."""
    m = copy.deepcopy(mech)
    m.reac_ptr, m.prod_ptr = mech.prod_ptr, mech.reac_ptr
    m.reac_sp, m.prod_sp = mech.prod_sp, mech.reac_sp
    m.reac_nu, m.prod_nu = mech.prod_nu, mech.reac_nu
    return m


def test_O4_reverse_reaction_identity_Kc(t3):
    """T3: R1 is R0 written backwards, so K_c(R0) K_c(R1) = 1 (Eq. 8-9)."""
    mech, batch, om = t3
    d = orc.detail(om, batch.T[0], batch.P[0], batch.Y[:, 0])
    assert close(d["Kc"][0] * d["Kc"][1], 1.0, 1e-14)


def test_O7_kf_over_kr_is_Kc_and_Kc_definition():
    """k_f/k_r = K_c (Eq. 7) with K_c from Eq. 8-9 evaluated here from the species thermo:
    K_c = exp(sum nu (s/R - h/RT)) (Patm/RT)^{sum nu}."""
    mech, batch = synth.make_config("C0", 8)
    om = oracle_mech(mech)
    for r in range(3):
        T = batch.T[r]
        d = orc.detail(om, T, batch.P[r], batch.Y[:, r])
        g = np.array([(lambda cp, h, s: s - h)(*orc.nasa7(mech.nasa[i], T)) for i in range(mech.n_species)])
        for k in range(mech.n_reactions):
            dg, dn = 0.0, 0
            for j in range(mech.prod_ptr[k], mech.prod_ptr[k + 1]):
                dg += mech.prod_nu[j] * g[mech.prod_sp[j]]
                dn += mech.prod_nu[j]
            for j in range(mech.reac_ptr[k], mech.reac_ptr[k + 1]):
                dg -= mech.reac_nu[j] * g[mech.reac_sp[j]]
                dn -= mech.reac_nu[j]
            Kc = np.exp(dg) * (PATM / (RGAS * T)) ** dn
            assert close(d["Kc"][k], Kc, 1e-12)
            assert close(d["kf"][k] / d["kr"][k], d["Kc"][k], 1e-14)


def test_O8_q_sign_flip_under_swap():
    """Swapping reactants and products while swapping k_f <-> k_r flips the sign of q.  The swapped
    mechanism gets k_f' := k_r by construction: K_c' = 1/K_c, so choose A' with k_f' = k_r; here we
    check the structural form on plain reactions: q'(k_f'=k_r, k_r'=k_f) = -q, through
    q' = k_f' prod C^{nu''} - k_r' prod C^{nu'}."""
    mech, batch = synth.make_config("C0", 4)
    plain = np.nonzero(mech.rtype == 0)[0]
    om, oms = oracle_mech(mech), oracle_mech(_swap(mech))
    for r in range(4):
        d = orc.detail(om, batch.T[r], batch.P[r], batch.Y[:, r])
        ds = orc.detail(oms, batch.T[r], batch.P[r], batch.Y[:, r])
        # swapped mechanism has the same A,b,Ea so k_f' = k_f and K_c' = 1/K_c:
        assert np.all(rel_err(ds["Kc"] * d["Kc"], np.ones_like(d["Kc"])) < 1e-13)
        # q' = kf (prodC'' - prodC' * Kc) = -Kc * q  (exact algebra) -> sign flips, magnitude scales by Kc
        assert np.all(rel_err(ds["q"][plain], -d["Kc"][plain] * d["q"][plain]) < 1e-9)
        assert np.all(np.sign(ds["q"][plain]) == -np.sign(d["q"][plain]))


@pytest.mark.parametrize("cfg,n", [("C0", 64), ("C1", 32), ("C2", 4), ("P5", 2)])
def test_O9_mass_conservation(cfg, n):
    """sum_k W_k wdot_k = 0 on element-balanced mechanisms, relative <= 1e-12 of sum |W_k wdot_k|."""
    mech, batch = synth.make_config(cfg, n)
    out = orc.evaluate(oracle_mech(mech), batch.T, batch.P, batch.Y, want=("wdot", "q"))
    ww = mech.W[:, None] * out["wdot"]
    # round-off scale: the individual reaction contributions, not the (possibly cancelling) wdot
    contrib = np.zeros_like(out["wdot"])
    for k in range(mech.n_reactions):
        for ptr, sp, nu in ((mech.reac_ptr, mech.reac_sp, mech.reac_nu), (mech.prod_ptr, mech.prod_sp, mech.prod_nu)):
            for j in range(ptr[k], ptr[k + 1]):
                contrib[sp[j]] += nu[j] * np.abs(out["q"][k]) * mech.W[sp[j]]
    assert np.all(np.abs(ww.sum(axis=0)) <= 1e-12 * contrib.sum(axis=0))
    # literal form of the north_star check wherever wdot does not itself cancel
    assert np.median(np.abs(ww.sum(axis=0)) / np.abs(ww).sum(axis=0)) <= 1e-12


def test_O6_lindemann_limits():
    """k -> k0 [M] as P_r -> 0 and k -> k_inf as P_r -> inf; exactly k/k_inf = Pr/(1+Pr)."""
    mech, batch = synth.toy_t3()
    for scale, Pr_expect in ((1e-12, "low"), (1e12, "high")):
        mm = copy.deepcopy(mech)
        mm.rtype = np.array([0, 1, 2], dtype=np.uint8)
        mm.A0 = mech.A0 * scale
        d = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])
        Pr, kf, kinf, k0, M = d["Pr"][2], d["kf"][2], d["kinf"][2], d["k0"][2], d["M"][2]
        assert close(kf / kinf, Pr / (1 + Pr), 1e-15)
        if Pr_expect == "low":
            assert Pr < 1e-11 and close(kf, k0 * M, 1e-11)
        else:
            assert Pr > 1e11 and close(kf, kinf, 1e-11)


def test_O6_troe_F_equals_Fcent_at_center_and_bounds():
    """At log10 P_r = -c the broadening factor is exactly F_cent (f1 = 0); F in [F_cent, 1]."""
    mech, batch = synth.toy_t3()
    om = oracle_mech(mech)
    d = orc.detail(om, batch.T[0], batch.P[0], batch.Y[:, 0])
    Fc, Pr = d["Fcent"][2], d["Pr"][2]
    c = -0.4 - 0.67 * np.log10(Fc)
    mm = copy.deepcopy(mech)
    mm.A0 = mech.A0 * (10.0 ** (-c) / Pr)
    d2 = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])
    assert close(d2["Pr"][2], 10.0 ** (-c), 1e-13)
    assert close(d2["F"][2], Fc, 1e-13)
    for s in 10.0 ** np.linspace(-10, 10, 41):
        mm.A0 = mech.A0 * s
        F = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])["F"][2]
        assert Fc * (1 - 1e-14) <= F <= 1.0


def test_O5_third_body_default_efficiency_and_falloff_list():
    """[M] = sum_i alpha_i C_i with alpha=1 unless listed; a falloff reaction honours a list (g7)."""
    mech, batch = synth.toy_t3()
    d = orc.detail(oracle_mech(mech), batch.T[0], batch.P[0], batch.Y[:, 0])
    C = d["C"]
    assert close(d["M"][0], C.sum(), 1e-15) and close(d["M"][2], C.sum(), 1e-15)
    assert close(d["M"][1], 2.5 * C[0] + C[1] + 0.7 * C[2], 1e-15)
    mm = copy.deepcopy(mech)
    mm.eff_ptr = np.array([0, 0, 2, 3], dtype=np.int32)
    mm.eff_sp = np.array([0, 2, 1], dtype=np.int32)
    mm.eff_val = np.array([2.5, 0.7, 3.0])
    d2 = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])
    assert close(d2["M"][2], C[0] + 3.0 * C[1] + C[2], 1e-15)
    assert close(d2["Pr"][2] / d["Pr"][2], d2["M"][2] / d["M"][2], 1e-14)


def test_O8_three_body_multiplies_both_directions(t3):
    """Reading g6: for rtype 1, q = [M] (kf prodC' - kr prodC''); falloff gets no extra [M]."""
    mech, batch, om = t3
    d = orc.detail(om, batch.T[0], batch.P[0], batch.Y[:, 0])
    C = d["C"]
    assert close(d["q"][1], d["M"][1] * (d["kf"][1] * C[2] - d["kr"][1] * C[0] * C[1]), 1e-14)
    assert close(d["q"][2], d["kf"][2] * C[0] * C[1] - d["kr"][2] * C[2], 1e-14)


def test_irreversible_reaction_has_zero_kr():
    mech, batch = synth.toy_t3()
    mm = copy.deepcopy(mech)
    mm.reversible = np.array([0, 1, 1], dtype=np.uint8)
    d = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])
    assert d["kr"][0] == 0.0 and close(d["q"][0], d["kf"][0] * d["C"][0] * d["C"][1], 1e-15)


def test_O8_integer_powers():
    """nu=2,3 by repeated multiplication equals C**nu; a reaction 2A + B <=> 3D."""
    mech, batch = synth.toy_t3()
    mm = copy.deepcopy(mech)
    mm.reac_nu = np.array([2, 1, 1, 1, 1], dtype=np.int32)  # R0: 2 S0 + S1
    mm.prod_nu = np.array([3, 1, 1, 1], dtype=np.int32)     # R0: 3 S2
    d = orc.detail(oracle_mech(mm), batch.T[0], batch.P[0], batch.Y[:, 0])
    C = d["C"]
    assert close(d["q"][0], d["kf"][0] * C[0] ** 2 * C[1] - d["kr"][0] * C[2] ** 3, 1e-14)
    # sum nu = 3 - 3 = 0 -> K_c = K_p
    assert close(d["Kc"][0], d["Kp"][0], 1e-15)


def test_O10_residual_sum_invariant():
    """sum_i F_i = (sum Y - sum Y_in)/tau because sum W wdot = 0."""
    mech, batch = synth.make_config("C1", 16)
    mech2, _ = synth.make_config("C2", 1)
    out = orc.evaluate(oracle_mech(mech), batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("F", "wdot"))
    lhs = out["F"].sum(axis=0)
    rhs = (batch.Y.sum(axis=0) - batch.Yin.sum(axis=0)) / batch.tau
    scale = np.abs(out["F"]).sum(axis=0)
    assert np.all(np.abs(lhs - rhs) <= 1e-12 * scale)
    # definition, retyped with numpy on the oracle's own wdot and an independently computed rho
    Wbar = 1.0 / (batch.Y / mech.W[:, None]).sum(axis=0)
    rho = batch.P * Wbar / (RGAS * batch.T)
    F = (batch.Y - batch.Yin) / batch.tau - out["wdot"] * mech.W[:, None] / rho
    assert np.all(rel_err(out["F"], F) < 1e-12)


# ------------------------------------------------------------------ brute force
@pytest.mark.parametrize("cfg,n", [("C0", 3), ("C1", 1)])
def test_whole_path_brute_force_mpmath(cfg, n):
    """Dense 50-digit evaluation of k_f, k_r, q, wdot, F vs the double oracle: <= 1e-13
    (q, wdot: relative to the round-off scale of their terms)."""
    mech, batch = synth.make_config(cfg, n)
    om = oracle_mech(mech)
    out = orc.evaluate(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("kf", "kr", "q", "wdot", "F"))
    for r in range(n):
        ref = mp_dense.evaluate(mech, batch.T[r], batch.P[r], batch.Y[:, r], batch.Yin[:, r], batch.tau[r])
        kf = np.array([float(x["kf"]) for x in ref["rx"]])
        kr = np.array([float(x["kr"]) for x in ref["rx"]])
        q = np.array([float(x["q"]) for x in ref["rx"]])
        assert rel_err(out["kf"][:, r], kf).max() < 1e-13
        assert rel_err(out["kr"][:, r], kr).max() < 1e-13
        # q may cancel: scale by |fwd|+|rev| ~ use max(|q|, tiny) relative with a cancellation allowance
        assert np.median(rel_err(out["q"][:, r], q)) < 1e-13 and rel_err(out["q"][:, r], q).max() < 1e-10
        w = np.array([float(x) for x in ref["wdot"]])
        big = np.abs(w) > 1e-12 * np.abs(w).max()
        assert rel_err(out["wdot"][big, r], w[big]).max() < 1e-10
        F = np.array([float(x) for x in ref["F"][1:]])
        assert rel_err(out["F"][:, r], F).max() < 1e-9


# ------------------------------------------------------------------ O11 Jacobian
def test_O11_T3_columns_long_double_and_double(t3):
    mech, batch, om = t3
    jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=True)
    jd = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=False)
    gold = np.array([GOLD["J_cols"][c] for c in ("T", "Y0", "Y1", "Y2")])  # [col][row]
    # long double: same floor law as 8(c)-J with eps = 2^-64 (noise 2000x lower than double);
    # golden printed to 12 digits
    Kj = np.array([1024.0, 32.0, 32.0, 32.0])
    floor_ld = 2.0 ** -64 * jl["S"][0][None, :] / jl["H"][0][:, None]
    assert np.all(np.abs(jl["J"][0] - gold) <= 1e-11 * np.abs(gold) + Kj[:, None] * floor_ld)
    # double: within the forward-difference round-off floor of 8(c)-J
    worst, fr_T, fr_Y = jacobian_floor_ratio(jd["J"], jl["J"], jl["S"], jl["H"])
    assert worst <= 1.0, (worst, fr_T, fr_Y)
    # h pinned: h_0 for T=1500
    assert jd["H"][0, 0] == float.fromhex("0x1.f751050000000p-17")
    assert np.array_equal(jd["H"], jl["H"])


def test_O11_invariants_row0_and_column_sums():
    """Row 0 of J is exactly e_0 (F_T = T - T_set, g13); species rows of a Y column sum to 1/tau and
    of the T column to 0 (mass conservation), up to the difference-quotient round-off floor."""
    mech, batch = synth.make_config("C4", 6)
    om = oracle_mech(mech)
    for ld in (False, True):
        j = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=ld)
        J = j["J"]  # [N][col][row]
        assert np.all(J[:, 0, 0] == 1.0) and np.all(J[:, 1:, 0] == 0.0)
        colsum = J[:, :, 1:].sum(axis=2)  # [N][col]
        floor = (64 * EPS if not ld else EPS) * j["S"][:, None, 1:].sum(axis=2) / j["H"]
        target = np.concatenate([np.zeros((batch.n, 1)), np.repeat(1.0 / batch.tau[:, None], mech.n_species, 1)], axis=1)
        assert np.all(np.abs(colsum - target) <= 1e-9 * np.abs(target) + floor)


def test_O11_double_within_floor_of_long_double_C4():
    mech, batch = synth.make_config("C4", 8)
    om = oracle_mech(mech)
    jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=True)
    jd = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=False)
    worst, fr_T, fr_Y = jacobian_floor_ratio(jd["J"], jl["J"], jl["S"], jl["H"])
    assert worst <= 1.0, (worst, fr_T, fr_Y)
    # the residuals themselves agree to ~1e-14
    assert np.all(np.abs(jd["F0"] - jl["F0"]) <= 1e-11 * np.maximum(np.abs(jl["F0"]), 1e-12 * np.abs(jl["F0"]).max(axis=1, keepdims=True)) + 1e-300)


def test_O11_linear_part_exact():
    """With all A = 0 (no chemistry) F_i = (Y_i - Yin_i)/tau: J[species block] = I/tau, T column 0."""
    mech, batch = synth.make_config("C0", 4)
    mm = copy.deepcopy(mech)
    mm.A = np.zeros_like(mech.A)
    j = orc.jacobian(oracle_mech(mm), batch.T, batch.P, batch.Y, batch.Yin, batch.tau)
    K = mech.n_species
    for r in range(4):
        Jr = j["J"][r].T  # [row][col]
        expect = np.zeros((K + 1, K + 1))
        expect[0, 0] = 1.0
        expect[1:, 1:] = np.eye(K) / batch.tau[r]
        # (Y+h - Yin)/tau - (Y - Yin)/tau over h: exact up to eps |Y - Yin|/tau / h
        tol = 4 * EPS * (np.abs(batch.Y[:, r] - batch.Yin[:, r]) / batch.tau[r])[:, None] / j["H"][r][None, 1:]
        assert np.all(np.abs(Jr[1:, 1:] - expect[1:, 1:]) <= tol + 1e-9 * expect[1:, 1:])
        assert np.all(Jr[1:, 0] == 0.0) and np.all(Jr[0] == expect[0])


def test_O11_roundoff_scale_S_against_its_definition(t3):
    """The floor term of every Jacobian criterion (tests/util.py: K_j eps S_i / h_j) rests on the scale S that
    jac_batch returns.  Pin it against SURVEY.md 8(c)-J's definition typed out independently at 50 digits
    (tests/mp_dense.py: dense nu', nu'', mp.power): T3 (plain, three-body and Troe reactions) with and without
    the energy row, and reactors of C0 (duplicates, efficiency lists) and C1 (every reaction type)."""
    mech, batch, om = t3
    for Tin in (None, 300.0):
        j = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau,
                         Tin=None if Tin is None else np.array([Tin]))
        S = mp_dense.roundoff_scale(mech, batch.T[0], batch.P[0], batch.Y[:, 0], batch.Yin[:, 0], batch.tau[0], Tin=Tin)
        assert j["S"][0, 0] == 0.0 if Tin is None else close(j["S"][0, 0], S[0], 1e-13)
        for i in range(1, 4):
            assert close(j["S"][0, i], S[i], 1e-13), (i, j["S"][0, i], S[i])
    for cfg, n in (("C0", 2), ("C1", 1)):
        mech, batch = synth.make_config(cfg, n)
        om = oracle_mech(mech)
        Tin = np.full(n, 350.0)
        for use_tin in (False, True):
            j = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin if use_tin else None)
            jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin if use_tin else None, long_double=True)
            for r in range(n):
                S = mp_dense.roundoff_scale(mech, batch.T[r], batch.P[r], batch.Y[:, r], batch.Yin[:, r], batch.tau[r],
                                            Tin=350.0 if use_tin else None)
                for i in range(mech.n_species + 1):
                    if i == 0 and not use_tin:
                        assert j["S"][r, 0] == 0.0 and jl["S"][r, 0] == 0.0
                        continue
                    assert close(j["S"][r, i], S[i], 1e-12), (cfg, r, i)
                    assert close(jl["S"][r, i], S[i], 1e-12), (cfg, r, i)


# ------------------------------------------------------------------ energy row
def test_energy_row_T3_golden_rederived_and_matched(t3):
    """Steady Eq. 3 as the residual F_T = -dT/dt: the T3 values printed in SURVEY.md 8(c)
    re-derived with mpmath, then the oracle against them."""
    mech, batch, om = t3
    g = GOLD["energy_Tin300"]
    m = mp_dense.evaluate(mech, batch.T[0], batch.P[0], batch.Y[:, 0], batch.Yin[:, 0], batch.tau[0], Tin=300.0)
    for i in range(3):
        assert close(m["h"][i], g["h_erg_per_g"][i], 1e-15)
    assert close(m["cp_mix"], g["cp_mix"], 1e-15) and close(m["FT"], g["F_T"], 1e-15)
    out = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, np.array([300.0]), batch.Yin, batch.tau)
    assert close(out["FT"][0], g["F_T"], 1e-12)
    for i in range(3):
        assert close(out["F"][i, 0], GOLD["F"][1 + i], 1e-12)          # species rows unchanged (O10)


def test_energy_row_vanishes_without_inflow_enthalpy_difference_or_reaction():
    """With every rate constant negligible (A -> 1e-300) and T_in = T the energy row is 0; with T_in != T it
    is the pure inflow term -(1/tau) sum Y_in (h_in - h) / cp_mix, linear in 1/tau."""
    mech, batch = synth.make_config("C0", 4)
    mech.A[:] = 1e-300
    om = oracle_mech(mech)
    same = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, batch.T, batch.Yin, batch.tau)
    assert np.all(np.abs(same["FT"]) <= 1e-250)
    Tin = np.full(4, 300.0)
    a = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, Tin, batch.Yin, batch.tau)
    b = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, Tin, batch.Yin, 2.0 * batch.tau)
    assert np.allclose(a["FT"], 2.0 * b["FT"], rtol=1e-13, atol=0)
    for r in range(4):
        hin = np.array([orc.nasa7(mech.nasa[i], 300.0)[1] * RGAS * 300.0 / mech.W[i] for i in range(mech.n_species)])
        h = np.array([orc.nasa7(mech.nasa[i], batch.T[r])[1] * RGAS * batch.T[r] / mech.W[i] for i in range(mech.n_species)])
        cp = sum(batch.Y[i, r] * orc.nasa7(mech.nasa[i], batch.T[r])[0] * RGAS / mech.W[i] for i in range(mech.n_species))
        expect = -(batch.Yin[:, r] @ (hin - h)) / batch.tau[r] / cp
        assert close(a["FT"][r], expect, 1e-12)


@pytest.mark.parametrize("cfg,n", [("C0", 3), ("C1", 1)])
def test_energy_row_brute_force_mpmath(cfg, n):
    """Whole adiabatic residual on generated mechanisms against the dense 50-digit evaluation."""
    mech, batch = synth.make_config(cfg, n)
    om = oracle_mech(mech)
    Tin = np.linspace(300.0, 600.0, n)
    out = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, Tin, batch.Yin, batch.tau)
    for r in range(n):
        m = mp_dense.evaluate(mech, batch.T[r], batch.P[r], batch.Y[:, r], batch.Yin[:, r], batch.tau[r], Tin=Tin[r])
        # the energy row is a difference of large terms: compare on the scale of its parts
        scale = max(abs(float(m["FT"])), 1e-12 * float(sum(abs(x) for x in m["h"])) / float(m["cp_mix"]) / float(batch.tau[r]))
        assert abs(out["FT"][r] - float(m["FT"])) <= 1e-10 * scale


def test_energy_row_long_double_agrees_with_double(t3):
    mech, batch, om = t3
    d = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, np.array([300.0]), batch.Yin, batch.tau)
    l = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, np.array([300.0]), batch.Yin, batch.tau, long_double=True)
    assert close(d["FT"][0], l["FT"][0], 1e-13)


def test_energy_jacobian_row0_against_exact_quotients_and_species_rows_unchanged(t3):
    """Adiabatic Jacobian on T3: row 0 (energy row) of every column against the exact difference quotient
    from 50-digit arithmetic with the double-precision step h_j (g15), inside the round-off floor of the
    method; rows 1..K are the species rows of the fixed-temperature Jacobian, bit for bit."""
    mech, batch, om = t3
    Tin = np.array([300.0])
    jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin, long_double=True)
    jd = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin)
    j0 = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau)
    assert np.array_equal(jd["J"][:, :, 1:], j0["J"][:, :, 1:])
    assert close(jd["F0"][0, 0], GOLD["energy_Tin300"]["F_T"], 1e-12)
    x = np.concatenate([batch.T, batch.Y[:, 0]])
    base = mp_dense.evaluate(mech, x[0], batch.P[0], x[1:], batch.Yin[:, 0], batch.tau[0], Tin=300.0)
    for j in range(4):
        delta = 1e-8 * max(abs(x[j]), 1e-10)
        xp = x.copy()
        xp[j] = x[j] + delta
        h = xp[j] - x[j]
        assert jl["H"][0, j] == h
        pert = mp_dense.evaluate(mech, xp[0], batch.P[0], xp[1:], batch.Yin[:, 0], batch.tau[0], Tin=300.0)
        exact = float((pert["FT"] - base["FT"]) / mpf(float(h)))
        floor = EPS * jl["S"][0, 0] / h
        assert abs(jl["J"][0, j, 0] - exact) <= 1e-9 * abs(exact) + 1.0 * floor, j      # 80-bit: well inside
        assert abs(jd["J"][0, j, 0] - exact) <= 1e-9 * abs(exact) + (1024.0 if j == 0 else 32.0) * floor, j


def test_energy_jacobian_double_within_floor_of_long_double_C4():
    mech, batch = synth.make_config("C4", 6)
    om = oracle_mech(mech)
    Tin = np.linspace(300.0, 650.0, 6)
    jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin, long_double=True)
    jd = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin)
    worst, fr_T, fr_Y = jacobian_floor_ratio(jd["J"], jl["J"], jl["S"], jl["H"])
    assert worst <= 1.0, (worst, fr_T, fr_Y)
    assert np.all(jl["S"][:, 0] > 0)


# ------------------------------------------------------------------ linear solve
def _colmajor(M):
    """[N][n][n] row-major matrices -> the J layout A[r, col, row]."""
    return np.ascontiguousarray(np.swapaxes(np.asarray(M, dtype=np.float64), 1, 2))


def test_lu_solve_exact_small_systems_and_row_exchange():
    from fractions import Fraction
    mats = [[[2, 1], [1, 3]], [[0, 2], [3, 1]],                       # the second needs a row exchange
            [[4, -2, 1], [-2, 4, -2], [1, -2, 4]], [[1, 2, 3], [4, 5, 6], [7, 8, 10]]]
    rhs = [[3, 5], [4, 5], [11, -16, 17], [6, 15, 25]]
    for M, b in zip(mats, rhs):
        n = len(b)
        # exact solution by Cramer-free rational elimination
        A = [[Fraction(v) for v in row] + [Fraction(bb)] for row, bb in zip(M, b)]
        for k in range(n):
            p = next(i for i in range(k, n) if A[i][k] != 0)
            A[k], A[p] = A[p], A[k]
            for i in range(n):
                if i != k:
                    f = A[i][k] / A[k][k]
                    A[i] = [u - f * v for u, v in zip(A[i], A[k])]
        exact = np.array([float(A[i][n] / A[i][i]) for i in range(n)])
        x, info = orc.lu_solve(_colmajor([M]), np.array([b], dtype=np.float64))
        assert info[0] == 0 and np.allclose(x[0], exact, rtol=1e-14, atol=0)


def test_lu_solve_reports_a_zero_pivot():
    x, info = orc.lu_solve(_colmajor([[[1, 2], [2, 4]], [[0, 0], [0, 1]]]), np.ones((2, 2)))
    assert info[0] == 2 and info[1] == 1


def test_lu_solve_matches_lapack_and_is_backward_stable():
    rng = np.random.default_rng(21)
    N, n = 16, 54
    M = rng.standard_normal((N, n, n)) + 4.0 * np.eye(n)
    b = rng.standard_normal((N, n))
    x, info = orc.lu_solve(_colmajor(M), b)
    assert np.all(info == 0)
    ref = np.linalg.solve(M, b[:, :, None])[:, :, 0]                    # LAPACK dgesv
    assert np.abs(x - ref).max() <= 1e-12 * np.abs(ref).max()
    res = np.abs(np.einsum("rij,rj->ri", M, x) - b).max(axis=1)
    bound = n * EPS * (np.abs(M).sum(axis=2).max(axis=1) * np.abs(x).max(axis=1) + np.abs(b).max(axis=1))
    assert np.all(res <= 8 * bound)
    xl, _ = orc.lu_solve(_colmajor(M), b, long_double=True)
    assert np.abs(x - xl).max() <= 1e-12 * np.abs(xl).max()


# ------------------------------------------------------------------ pseudo-transient step
def test_ptc_step_exact_rational_and_scalar_closed_form():
    """(I/dt + J) dx = -F (implicit Euler on dx/dt = -F).  Expected values by exact rational
    arithmetic on the shifted system, written out here; the scalar case is dx = -F/(1/dt + J)."""
    from fractions import Fraction
    J = [[2, 1], [1, 3]]
    F = [3, 5]
    dt = Fraction(1, 2)                              # 1/dt = 2 -> A = [[4, 1], [1, 5]], b = (-3, -5)
    det = Fraction(4 * 5 - 1 * 1)
    exact = [float((Fraction(-3) * 5 - Fraction(-5) * 1) / det), float((Fraction(4) * -5 - Fraction(1) * -3) / det)]
    assert exact == [float(Fraction(-10, 19)), float(Fraction(-17, 19))]
    dx, info = orc.ptc_step(_colmajor([J]), np.array([F], dtype=np.float64), np.array([float(dt)]))
    assert info[0] == 0 and np.allclose(dx[0], exact, rtol=1e-15, atol=0)
    # scalar systems: dx = -F / (1/dt + J)
    Js = np.array([[[3.0]], [[-0.25]], [[1e6]]])
    Fs = np.array([[2.0], [1.0], [-4.0]])
    dts = np.array([0.5, 2.0, 1e-3])
    dx, info = orc.ptc_step(Js, Fs, dts)
    want = -Fs[:, 0] / (1.0 / dts + Js[:, 0, 0])
    assert np.all(info == 0) and np.allclose(dx[:, 0], want, rtol=2e-16 * 4, atol=0)
    # a transposed operand would show here: non-symmetric J
    Jn = [[1, 4], [0, 1]]                            # dt = 1: A = [[2, 4], [0, 2]], b = (-2, -2) -> dx = (1, -1)
    dx, _ = orc.ptc_step(_colmajor([Jn]), np.array([[2.0, 2.0]]), np.array([1.0]))
    assert np.array_equal(dx[0], [1.0, -1.0])


def test_ptc_step_limits_newton_and_explicit_euler():
    rng = np.random.default_rng(44)
    N, n = 8, 54
    M = rng.standard_normal((N, n, n)) + 4.0 * np.eye(n)
    F = rng.standard_normal((N, n))
    # dt = inf: the shift vanishes and the step is the Newton step J dx = -F (NEXT-2's solve, LAPACK here)
    dx, info = orc.ptc_step(_colmajor(M), F, np.full(N, np.inf))
    newton = np.linalg.solve(M, -F[:, :, None])[:, :, 0]
    assert np.all(info == 0) and np.abs(dx - newton).max() <= 1e-12 * np.abs(newton).max()
    # dt -> 0: (I/dt + J)^-1 = dt (I - dt J + ...), so dx = -dt F + dt^2 J F + O(dt^3)
    dt = np.full(N, 1e-7)
    dx, _ = orc.ptc_step(_colmajor(M), F, dt)
    euler = -dt[:, None] * F
    second = dt[:, None] ** 2 * np.einsum("rij,rj->ri", M, F)
    assert np.abs(dx - euler).max() <= 2e-7 * 60 * np.abs(euler).max()       # |dt J| ~ 1e-7 * ||J||
    assert np.abs(dx - (euler + second)).max() <= 1e-11 * np.abs(euler).max()
    # general dt against LAPACK on the shifted matrix, plus a system the shift makes singular
    dt = 10.0 ** rng.uniform(-4, 1, N)
    dx, info = orc.ptc_step(_colmajor(M), F, dt)
    ref = np.linalg.solve(M + np.eye(n)[None] / dt[:, None, None], -F[:, :, None])[:, :, 0]
    assert np.all(info == 0) and np.abs(dx - ref).max() <= 1e-12 * np.abs(ref).max()
    _, info = orc.ptc_step(np.array([[[-2.0]]]), np.array([[1.0]]), np.array([0.5]))   # 1/dt + J = 0
    assert info[0] == 1


# ------------------------------------------------------------------ hybrid Newton / pseudo-transient solver (NEXT-4)
def _two_species(rx, W, A, b=0.0, Ea=5e3, a6B=3.0):
    """One reversible reaction between two species (inputs only; a6 of the second species sets the equilibrium)."""
    nasa = np.array([[3.5, 1e-4, 0.0, 0.0, 0.0, -1000.0, 2.0],
                     [3.9, 3e-4, -2e-8, 0.0, 0.0, -1600.0, a6B]])
    reac_ptr, reac_sp, reac_nu = synth._side_csr([rx[0]])
    prod_ptr, prod_sp, prod_nu = synth._side_csr([rx[1]])
    return synth.Mechanism(
        n_species=2, n_reactions=1, atoms=np.zeros((2, 4), dtype=np.int32), W=np.array(W, dtype=np.float64), nasa=nasa,
        A=np.array([A]), b=np.array([b]), Ea=np.array([Ea]), rtype=np.zeros(1, dtype=np.uint8),
        reversible=np.ones(1, dtype=np.uint8), reac_ptr=reac_ptr, reac_sp=reac_sp, reac_nu=reac_nu,
        prod_ptr=prod_ptr, prod_sp=prod_sp, prod_nu=prod_nu, eff_ptr=np.zeros(2, dtype=np.int32),
        eff_sp=np.zeros(0, dtype=np.int32), eff_val=np.zeros(0), A0=np.zeros(1), b0=np.zeros(1), Ea0=np.zeros(1),
        troe=np.zeros((1, 4)), meta={"name": "two-species"})


def test_solver_inert_mechanism_reaches_the_inlet_composition_in_one_newton_step():
    """Without chemistry F = (Y - Y_in)/tau is linear: one Newton step lands on Y = Y_in up to the accuracy of the
    forward-difference Jacobian (eps |Y - Y_in| / h ~ 1e-8 relative), the next iteration's correction is that
    small and passes a 1e-6 tolerance test (2 Newton iterations, no pseudo-transient step), and has refined the
    estimate to round-off."""
    mech, batch = synth.make_config("C0", 12)
    mm = copy.deepcopy(mech)
    mm.A = np.zeros_like(mech.A)
    om = oracle_mech(mm)
    one = orc.solve_hybrid(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, atol=1e-9, rtol=1e-6, max_iter=1)
    assert np.all(one["status"] == 1) and np.all(one["n_newton"] == 1)
    assert np.abs(one["Y"] - batch.Yin).max() <= 1e-6 * np.abs(batch.Y - batch.Yin).max()
    r = orc.solve_hybrid(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, atol=1e-9, rtol=1e-6)
    assert np.all(r["status"] == 0) and np.all(r["n_newton"] == 2) and np.all(r["n_ptc"] == 0)
    assert np.allclose(r["Y"], batch.Yin, rtol=1e-12, atol=1e-15) and np.array_equal(r["T"], batch.T)


def test_solver_isomerisation_closed_form_steady_state():
    """A <=> B with equal molar masses: wdot_A W/rho = -(k_f Y_A - k_r Y_B) whatever rho is, so the steady
    residual is LINEAR in Y and has the closed-form root
        Y_A = (Y_A,in / tau + k_r S) / (1/tau + k_f + k_r),  S = Y_A,in + Y_B,in,
    with k_f from Eq. 6 and k_r = k_f / K_c (Eq. 7-9, sum nu = 0) evaluated here with mpmath.  Newton on a linear
    residual converges in one step (+ one to confirm, which also removes the forward-difference error)."""
    from mpmath import exp as mexp, log as mlog, power as mpow
    mech = _two_species(((0,), (1,)), W=[28.0, 28.0], A=3.0e3, b=0.3, Ea=4.0e3)
    T, P, tau = 1400.0, 2.0 * PATM, 2e-3
    Yin = np.array([[0.7], [0.3]])
    Y0 = np.array([[0.2], [0.8]])
    r = orc.solve_hybrid(oracle_mech(mech), np.array([T]), np.array([P]), Y0, Yin, np.array([tau]), atol=1e-9, rtol=1e-6)
    Tm = mpf(T)
    kf = mpf(float(mech.A[0])) * mpow(Tm, mpf(float(mech.b[0]))) * mexp(-mpf(float(mech.Ea[0])) / (mp_dense.RCAL * Tm))
    def g(a):
        a = [mpf(float(v)) for v in a]
        hRT = a[0] + a[1] * Tm / 2 + a[2] * Tm**2 / 3 + a[3] * Tm**3 / 4 + a[4] * Tm**4 / 5 + a[5] / Tm
        sR = a[0] * mlog(Tm) + a[1] * Tm + a[2] * Tm**2 / 2 + a[3] * Tm**3 / 3 + a[4] * Tm**4 / 4 + a[6]
        return sR - hRT
    Kc = mexp(g(mech.nasa[1]) - g(mech.nasa[0]))
    kr = kf / Kc
    yA = (mpf("0.7") / mpf(tau) + kr) / (1 / mpf(tau) + kf + kr)
    assert r["status"][0] == 0 and r["n_newton"][0] == 2 and r["n_ptc"][0] == 0
    assert close(r["Y"][0, 0], yA, 1e-10) and close(r["Y"][1, 0], 1 - yA, 1e-10)
    assert 0.05 < float(yA) < 0.95 and abs(float(yA) - 0.7) > 0.05     # chemistry matters in this case


def _dimerisation_root(mech, T, P, Yin, tau):
    """Root of the steady residual of 2A <=> B (W_B = 2 W_A) with mpmath: Y_A + Y_B = 1 at steady state, so
    F_A(y) = 0 in one unknown, the residual taken from the dense 50-digit restatement (mp_dense)."""
    from mpmath import findroot
    def FA(y):
        return mp_dense.evaluate(mech, T, P, [y, 1 - y], Yin=Yin, tau=tau)["F"][1]
    return findroot(FA, (mpf("1e-6"), mpf("0.999999")), solver="illinois", maxsteps=400, verify=False)


def test_solver_nonlinear_root_and_the_switch_to_pseudo_transient():
    """2A <=> B (second order): the converged estimate is the root computed independently with mpmath.  From a
    good guess Newton alone converges; from a guess whose Newton trial leaves the admissible region
    (Y < -y_floor) the estimate is first conditioned by pseudo-transient steps (whole stages of max_ptc steps),
    then Newton converges to the same root; a budget too small is reported as not converged."""
    mech = _two_species(((0, 0), (1,)), W=[15.0, 30.0], A=2.0e9, b=0.0, Ea=2.0e3, a6B=23.0)
    T, P, tau = 1200.0, PATM, 1e-3
    Yin = np.array([[0.9], [0.1]])
    root = _dimerisation_root(mech, T, P, Yin[:, 0], tau)
    om = oracle_mech(mech)
    args = (np.array([T]), np.array([P]))
    good = orc.solve_hybrid(om, *args, np.array([[float(root) * 1.05], [1 - float(root) * 1.05]]), Yin, np.array([tau]),
                            atol=1e-14, rtol=1e-10, max_newton=20)
    assert good["status"][0] == 0 and good["n_ptc"][0] == 0 and 2 <= good["n_newton"][0] <= 8
    assert close(good["Y"][0, 0], root, 1e-8) and close(good["Y"][1, 0], 1 - root, 1e-8)
    # far guess: the first Newton trial is not admissible -> pseudo-transient conditioning -> Newton
    far = orc.solve_hybrid(om, *args, np.array([[1.0 - 1e-9], [1e-9]]), Yin, np.array([tau]), atol=1e-14, rtol=1e-10,
                           max_iter=400, max_newton=6, max_ptc=10, dt0=1e-9, dt_grow=2.0, dt_shrink=0.25, y_floor=0.0)
    bad = orc.solve_hybrid(om, *args, np.array([[1.0 - 1e-9], [1e-9]]), Yin, np.array([tau]), atol=1e-14, rtol=1e-10,
                           max_iter=100, max_newton=100, max_ptc=0 + 1, dt0=1e-30, dt_grow=1.0, y_floor=0.0)
    assert far["status"][0] == 0 and far["n_ptc"][0] > 0 and far["n_ptc"][0] % 10 == 0
    assert close(far["Y"][0, 0], root, 1e-8)
    assert far["n_newton"][0] + far["n_ptc"][0] <= 400
    # (with a vanishing pseudo-time step the estimate cannot move: Newton keeps failing from the same point)
    assert bad["status"][0] == 1 and bad["n_newton"][0] + bad["n_ptc"][0] == 100
    short = orc.solve_hybrid(om, *args, np.array([[0.5], [0.5]]), Yin, np.array([tau]), atol=1e-14, rtol=1e-10, max_iter=1)
    assert short["status"][0] == 1 and short["n_newton"][0] == 1 and short["n_ptc"][0] == 0


def test_solver_pseudo_transient_steps_with_a_huge_dt_are_newton_steps():
    """(I/dt + J) dx = -F tends to the Newton system as dt -> inf: a run that is forced through pseudo-transient
    stages (max_newton = 1) with dt0 = 1e300 walks through the same estimates as the pure Newton iteration.
    Tolerances are set so that neither run stops early."""
    mech = _two_species(((0, 0), (1,)), W=[15.0, 30.0], A=2.0e9, b=0.0, Ea=2.0e3, a6B=23.0)
    om = oracle_mech(mech)
    T, P, tau = np.array([1200.0]), np.array([PATM]), np.array([1e-3])
    Yin, Y0 = np.array([[0.9], [0.1]]), np.array([[0.55], [0.45]])
    for budget in (1, 2, 3, 4):
        kw = dict(atol=1e-300, rtol=1e-300, max_iter=budget, y_floor=np.inf)
        a = orc.solve_hybrid(om, T, P, Y0, Yin, tau, max_newton=100, **kw)
        b = orc.solve_hybrid(om, T, P, Y0, Yin, tau, max_newton=1, max_ptc=100, dt0=1e300, dt_grow=1.0, **kw)
        assert a["n_newton"][0] == budget and b["n_newton"][0] == 1 and b["n_ptc"][0] == budget - 1
        assert np.allclose(a["Y"], b["Y"], rtol=1e-12, atol=0)


def test_solver_adiabatic_inert_reactor_settles_at_the_inlet_state():
    """Energy row as row 0 (Tin given), no chemistry: the steady state is Y = Y_in, T = T_in (the inflow enthalpy
    difference sum Y_in (h_in - h(T)) vanishes only there, h being monotone in T)."""
    mech, batch = synth.make_config("C0", 6)
    mm = copy.deepcopy(mech)
    mm.A = np.zeros_like(mech.A)
    Tin = np.linspace(600.0, 900.0, 6)
    r = orc.solve_hybrid(oracle_mech(mm), batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin, atol=1e-12, rtol=1e-10,
                         max_newton=30, y_floor=np.inf)
    assert np.all(r["status"] == 0) and np.all(r["n_ptc"] == 0)
    assert np.allclose(r["T"], Tin, rtol=1e-9) and np.allclose(r["Y"], batch.Yin, rtol=1e-10, atol=1e-14)
