"""Parity of the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Tolerances (BASELINE.json: north_star): max relative error <= 1e-10 on
k_f, k_r, q and on wdot wherever |wdot| > 1e-12 max|wdot| (per reactor); <= 1e-9 on the residual
(relative to max(|F_i|, 1e-12 max_i|F_i|)); Jacobian by the floor criterion of SURVEY.md 8(c)-J
against the long-double oracle J*.
"""
import copy
import json
import os
from pathlib import Path

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2005_11468_b200 import synth
from util import floor_criterion, jacobian_floor_ratio, oracle_mech, rel_err, residual_rel_err, wdot_masked_rel_err

pytestmark = pytest.mark.gpu

TOL_K = 1e-10
RGAS = 8.31446261815324e7
TOL_F = 1e-9


@pytest.fixture(scope="module")
def torch_cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def binding(torch_cuda):
    from paper_2005_11468_b200 import binding as b
    b.lib()
    return b


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_eval(torch, binding, mech, batch, want_F=True):
    gm = binding.Mechanism.from_synth(mech)
    T, P, Y = dev(torch, batch.T), dev(torch, batch.P), dev(torch, batch.Y)
    kf, kr = gm.eval_kf_kr(T, P, Y)
    wdot, q = gm.eval_wdot(T, P, Y, want_q=True)
    out = dict(kf=kf.cpu().numpy(), kr=kr.cpu().numpy(), q=q.cpu().numpy(), wdot=wdot.cpu().numpy())
    if want_F:
        Yin, tau = dev(torch, batch.Yin), dev(torch, batch.tau)
        F, w2 = gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
        out["F"] = F.cpu().numpy()
        out["wdot_from_residual"] = w2.cpu().numpy()
    torch.cuda.synchronize()
    gm.close()
    return out


def check_against_oracle(mech, batch, got, q_tol=TOL_K):
    ref = orc.evaluate(oracle_mech(mech), batch.T, batch.P, batch.Y, batch.Yin, batch.tau,
                       want=("kf", "kr", "q", "wdot", "F"))
    assert rel_err(got["kf"], ref["kf"]).max() <= TOL_K
    assert rel_err(got["kr"], ref["kr"]).max() <= TOL_K
    # q = fwd - rev can cancel; the tolerance applies relative to the larger of |q| and 1e-12 of the
    # reactor's largest |q| (same masking rule as wdot)
    qerr, _ = wdot_masked_rel_err(got["q"], ref["q"])
    assert qerr.max() <= q_tol
    werr, mask = wdot_masked_rel_err(got["wdot"], ref["wdot"])
    assert mask.any() and werr.max() <= TOL_K
    if "F" in got:
        assert residual_rel_err(got["F"], ref["F"]).max() <= TOL_F
        assert np.array_equal(got["wdot_from_residual"], got["wdot"])
    return ref


# ------------------------------------------------------------------ configs
def test_C0_full_kf_kr_q_wdot(torch_cuda, binding):
    mech, batch = synth.make_config("C0")
    got = gpu_eval(torch_cuda, binding, mech, batch)
    check_against_oracle(mech, batch, got)


@pytest.mark.parametrize("cfg,n", [("C1", 2000), ("C2", 333), ("C3", 97), ("P5", 150)])
def test_configs_ragged_batches(torch_cuda, binding, cfg, n):
    """Several tiles plus a ragged tail (n not a multiple of 32), all reaction types."""
    mech, batch = synth.make_config(cfg, n)
    got = gpu_eval(torch_cuda, binding, mech, batch)
    check_against_oracle(mech, batch, got)


@pytest.mark.parametrize("K,I,tb,troe,n,expect", [
    (230, 900, 70, 60, 5 * 148 * 32 // 16 + 19, dict(eval_kernel=2, eval_acc_global=1)),   # tile copy in tensor memory, sums in L2
    (127, 100, 8, 6, 333, dict(eval_kernel=1)),                                             # resident kernel, K + 2 > 128: no copy
    (96, 700, 50, 40, 333, dict(eval_kernel=2, eval_acc_global=0)),                        # streamed parts, sums in shared memory
])
def test_kernel_variants_between_the_configs(torch_cuda, binding, K, I, tb, troe, n, expect):
    """The BASELINE configs land on four of the evaluation kernels' variants (resident with the tensor-memory copy: C1;
    streamed with tile and sums in tensor memory: C2; streamed without tensor memory, sums in L2: C3; sums in shared
    memory: P5).  Mechanisms sized to take the others, against the oracle like every config, and with the
    tensor-memory switch off."""
    torch = torch_cuda
    mech = synth.make_mechanism(n_species=K, n_reactions=I, n_third_body=tb, n_troe=troe, seed=4242 + K, mmax=3)
    batch = synth.make_states(K, n, seed=99 + K)
    gm = binding.Mechanism.from_synth(mech)
    info = gm.info()
    for k, v in expect.items():
        assert info[k] == v, (k, info)
    gm.close()
    got = gpu_eval(torch, binding, mech, batch)
    check_against_oracle(mech, batch, got)
    gm = binding.Mechanism.from_synth(mech)
    T, P, Y, Yin, tau = (dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
    F0, w0 = gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
    gm.set_option(binding.OPT_NO_TMEM, 1)
    F1, w1 = gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
    assert torch.equal(F0, F1) and torch.equal(w0, w1)
    gm.close()


def test_T3_goldens_direct(torch_cuda, binding):
    """The GPU path against the paper-derived T3 values themselves (tests/golden/t3_pins.json)."""
    gold = json.loads((Path(__file__).parent / "golden" / "t3_pins.json").read_text())
    mech, batch = synth.toy_t3()
    got = gpu_eval(torch_cuda, binding, mech, batch)
    for k, name in enumerate(("R0", "R1", "R2")):
        assert abs(got["kf"][k, 0] / gold[name]["kf"] - 1) <= 1e-12
        assert abs(got["kr"][k, 0] / gold[name]["kr"] - 1) <= 1e-12
        assert abs(got["q"][k, 0] / gold[name]["q"] - 1) <= 1e-11
    for i in range(3):
        assert abs(got["wdot"][i, 0] / (gold["wdot_sign"][i] * gold["wdot_abs"]) - 1) <= 1e-11
        assert abs(got["F"][i, 0] / gold["F"][i + 1] - 1) <= 1e-11


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("n", [1, 31, 32, 33, 64])
def test_tile_boundaries(torch_cuda, binding, n):
    mech, batch = synth.make_config("C1", n)
    got = gpu_eval(torch_cuda, binding, mech, batch)
    check_against_oracle(mech, batch, got)


def test_empty_batch_is_ok(torch_cuda, binding):
    torch = torch_cuda
    mech, _ = synth.make_config("C0", 1)
    gm = binding.Mechanism.from_synth(mech)
    z = torch.empty(0, dtype=torch.float64, device="cuda")
    Y = torch.empty((mech.n_species, 0), dtype=torch.float64, device="cuda")
    w = gm.eval_wdot(z, z, Y)
    assert w.shape == (mech.n_species, 0)
    gm.close()


def test_leading_dimension_larger_than_N(torch_cuda, binding):
    torch = torch_cuda
    mech, batch = synth.make_config("C1", 100)
    gm = binding.Mechanism.from_synth(mech)
    ld = 160
    Ybig = torch.full((mech.n_species, ld), float("nan"), dtype=torch.float64, device="cuda")
    Ybig[:, :100] = dev(torch, batch.Y)
    wbig = torch.full((mech.n_species, ld), -7.0, dtype=torch.float64, device="cuda")
    gm.eval_wdot(dev(torch, batch.T), dev(torch, batch.P), Ybig[:, :100], wdot=wbig[:, :100])
    ref = orc.evaluate(oracle_mech(mech), batch.T, batch.P, batch.Y, want=("wdot",))
    w = wbig.cpu().numpy()
    werr, _ = wdot_masked_rel_err(w[:, :100], ref["wdot"])
    assert werr.max() <= TOL_K
    assert np.all(w[:, 100:] == -7.0)  # padding untouched
    # psr_eval_residual / psr_eval_residual_energy take ONE ld for Y, Yin, F and wdot: outputs the binding
    # allocates must share it (a dense [K][N] tensor would be overrun), outputs the caller passes are checked
    Yinbig = torch.full((mech.n_species, ld), float("nan"), dtype=torch.float64, device="cuda")
    Yinbig[:, :100] = dev(torch, batch.Yin)
    T, P, tau, Tin = dev(torch, batch.T), dev(torch, batch.P), dev(torch, batch.tau), torch.full((100,), 300.0, dtype=torch.float64, device="cuda")
    refF = orc.evaluate(oracle_mech(mech), batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("wdot", "F"))
    Fbig = torch.full((mech.n_species, ld), -7.0, dtype=torch.float64, device="cuda")
    w2big = torch.full((mech.n_species, ld), -7.0, dtype=torch.float64, device="cuda")
    gm.eval_residual(T, P, Ybig[:, :100], Yinbig[:, :100], tau, F=Fbig[:, :100], wdot=w2big[:, :100])
    Fa, wa = gm.eval_residual(T, P, Ybig[:, :100], Yinbig[:, :100], tau, want_wdot=True)   # binding-allocated
    assert Fa.stride(0) == ld and wa.stride(0) == ld
    Fe, FTe, we = gm.eval_residual_energy(T, P, Ybig[:, :100], Tin, Yinbig[:, :100], tau, want_wdot=True)
    assert Fe.stride(0) == ld and we.stride(0) == ld
    Fe2 = torch.full((mech.n_species, ld), -7.0, dtype=torch.float64, device="cuda")
    gm.eval_residual_energy(T, P, Ybig[:, :100], Tin, Yinbig[:, :100], tau, F=Fe2[:, :100])
    torch.cuda.synchronize()
    for Fx in (Fbig[:, :100], Fa, Fe, Fe2[:, :100]):
        assert residual_rel_err(Fx.cpu().numpy(), refF["F"]).max() <= TOL_F
    for wx in (w2big[:, :100], wa):
        assert np.array_equal(wx.cpu().numpy(), w[:, :100])
    assert wdot_masked_rel_err(we.cpu().numpy(), w[:, :100])[0].max() <= 1e-11   # fused kernel vs warp-specialised one
    for big in (Fbig, w2big, Fe2):
        assert bool((big[:, 100:] == -7.0).all())  # padding untouched
    dense = torch.empty((mech.n_species, 100), dtype=torch.float64, device="cuda")
    for kw in (dict(F=dense), dict(wdot=dense)):
        with pytest.raises(ValueError):
            gm.eval_residual(T, P, Ybig[:, :100], Yinbig[:, :100], tau, **kw)
        with pytest.raises(ValueError):
            gm.eval_residual_energy(T, P, Ybig[:, :100], Tin, Yinbig[:, :100], tau, **kw)
    with pytest.raises(ValueError):
        gm.eval_residual(T, P, Ybig[:, :100], dev(torch, batch.Yin), tau)
    gm.close()


def _variant(mech, **kw):
    m = copy.deepcopy(mech)
    for k, v in kw.items():
        setattr(m, k, v)
    return m


def test_lindemann_irreversible_and_falloff_efficiencies(torch_cuda, binding):
    """Degenerate / rarely used branches: rtype 2, reversible = 0, efficiency list on a falloff
    reaction (reading g7), nu = 3."""
    mech, batch = synth.make_config("C1", 70)
    rtype = mech.rtype.copy()
    troe_idx = np.nonzero(rtype == 3)[0]
    rtype[troe_idx[::2]] = 2                      # half the Troe reactions become Lindemann
    reversible = mech.reversible.copy()
    reversible[::7] = 0
    # give the first Troe/Lindemann reactions an efficiency list
    eff_ptr, eff_sp, eff_val = [0], [], []
    old_ptr = mech.eff_ptr
    for k in range(mech.n_reactions):
        sp = list(mech.eff_sp[old_ptr[k]:old_ptr[k + 1]])
        val = list(mech.eff_val[old_ptr[k]:old_ptr[k + 1]])
        if k in troe_idx[:6]:
            sp, val = [1, 5, 9], [0.3, 2.0, 11.5]
        eff_sp += sp
        eff_val += val
        eff_ptr.append(len(eff_sp))
    m2 = _variant(mech, rtype=rtype, reversible=reversible, eff_ptr=np.array(eff_ptr, dtype=np.int32),
                  eff_sp=np.array(eff_sp, dtype=np.int32), eff_val=np.array(eff_val))
    got = gpu_eval(torch_cuda, binding, m2, batch)
    ref = check_against_oracle(m2, batch, got)
    assert np.all(got["kr"][::7] == 0.0) and np.all(ref["kr"][::7] == 0.0)


def test_long_factor_lists_and_nu3(torch_cuda, binding):
    """A reaction with more than 8 concentration factors takes the pooled-list path; nu = 3."""
    mech, batch = synth.make_config("C0", 40)
    m = copy.deepcopy(mech)
    # reaction 0: 3 A + 3 B + 2 C <=> 3 D + 3 E  (8 + 6 = 14 factors), not element balanced -- irrelevant here
    rp, rs, rn = list(m.reac_ptr), list(m.reac_sp), list(m.reac_nu)
    pp, ps, pn = list(m.prod_ptr), list(m.prod_sp), list(m.prod_nu)
    n_old_r, n_old_p = rp[1] - rp[0], pp[1] - pp[0]
    rs[rp[0]:rp[1]] = [0, 1, 2]
    rn[rp[0]:rp[1]] = [3, 3, 2]
    ps[pp[0]:pp[1]] = [3, 4]
    pn[pp[0]:pp[1]] = [3, 3]
    rp = [0] + [x + (3 - n_old_r) for x in rp[1:]]
    pp = [0] + [x + (2 - n_old_p) for x in pp[1:]]
    m.reac_ptr, m.reac_sp, m.reac_nu = (np.array(x, dtype=np.int32) for x in (rp, rs, rn))
    m.prod_ptr, m.prod_sp, m.prod_nu = (np.array(x, dtype=np.int32) for x in (pp, ps, pn))
    m.A = m.A.copy()
    m.A[0] = 1e40  # keep the 8th-order term visible next to the others
    got = gpu_eval(torch_cuda, binding, m, batch)
    check_against_oracle(m, batch, got)


def test_negative_and_zero_pre_exponentials(torch_cuda, binding):
    """Any finite A is valid input: a duplicate pair with a negative pre-exponential, A = 0 (a
    zero-rate reaction), on plain, three-body and Lindemann reactions, and a negative A and A0 together on Troe
    reactions (P_r stays positive).  Where the definition gives no number -- A0 <= 0 or A = 0 on a Troe reaction:
    log10 P_r of a non-positive P_r -- both sides must give NaN."""
    torch = torch_cuda
    mech, batch = synth.make_config("C1", 150)
    m = copy.deepcopy(mech)
    rt = np.asarray(m.rtype)
    plain, tb, troe = np.flatnonzero(rt == 0), np.flatnonzero(rt == 1), np.flatnonzero(rt == 3)
    m.A = m.A.copy(); m.A0 = m.A0.copy(); m.rtype = m.rtype.copy()
    m.A[plain[0]] *= -1.0          # negative pre-exponential (CHEMKIN duplicate)
    m.A[plain[1]] = 0.0            # zero-rate reaction
    m.A[tb[0]] *= -0.5
    m.A[tb[1]] = 0.0
    m.rtype[troe[0]] = 2           # Lindemann: k_inf < 0, k_0 > 0 (P_r < 0 is a number there)
    m.A[troe[0]] *= -1.0
    m.rtype[troe[1]] = 2           # Lindemann with A0 = 0: k_f = 0
    m.A0[troe[1]] = 0.0
    m.A[troe[2]] *= -1.0           # Troe, both negative: P_r > 0, k_f < 0
    m.A0[troe[2]] *= -1.0
    got = gpu_eval(torch, binding, m, batch)
    ref = check_against_oracle(m, batch, got)
    assert np.all(got["kf"][plain[0]] < 0) and np.all(got["kf"][plain[1]] == 0) and np.all(got["q"][plain[1]] == 0)
    assert np.all(got["kf"][troe[2]] < 0) and np.all(got["kf"][troe[1]] == 0)
    assert np.array_equal(np.sign(got["kr"]), np.sign(ref["kr"]))
    # no number by the definition: NaN on both sides, and only there
    m2 = copy.deepcopy(mech)
    m2.A = m2.A.copy(); m2.A0 = m2.A0.copy()
    m2.A0[troe[0]] = 0.0
    m2.A0[troe[1]] *= -1.0
    m2.A[troe[2]] = 0.0
    sub = batch.take(np.arange(40))
    got2 = gpu_eval(torch, binding, m2, sub, want_F=False)
    ref2 = orc.evaluate(oracle_mech(m2), sub.T, sub.P, sub.Y, want=("kf", "kr", "q", "wdot"))
    for name in ("kf", "q", "wdot"):
        assert np.array_equal(np.isnan(got2[name]), np.isnan(ref2[name])), name
    assert np.isnan(ref2["kf"][troe[:3]]).all() and not np.isnan(ref2["kf"][plain]).any()
    ok = ~np.isnan(ref2["kf"])
    assert rel_err(got2["kf"][ok], ref2["kf"][ok]).max() <= TOL_K


def test_negative_and_zero_mass_fractions_propagate(torch_cuda, binding):
    """Newton iterates may leave [0,1]; products by multiplication keep the sign."""
    mech, batch = synth.make_config("C1", 64)
    Y = batch.Y.copy()
    Y[3, :] = 0.0
    Y[7, ::2] *= -1e-3
    b2 = synth.ReactorBatch(batch.T, batch.P, Y, batch.Yin, batch.tau)
    got = gpu_eval(torch_cuda, binding, mech, b2)
    check_against_oracle(mech, b2, got)


def test_out_of_range_exp_arguments_take_the_library_path(torch_cuda, binding):
    """A few very cold reactors push exp arguments beyond |x| = 700 (Ea/RT ~ 1000).  The kernel's table
    exp is not valid there: the CTA must notice and repeat its reaction phase with the library exp, for
    every lane of the tile.  Warm lanes of the same tiles must still match the oracle to tolerance; in
    the cold lanes k_f (T-only, Eq. 6) must underflow the way the oracle's does."""
    torch = torch_cuda
    mech, batch = synth.make_config("C1", 96)
    T = batch.T.copy()
    cold = np.array([5, 40, 41, 95])
    T[cold] = [20.0, 25.0, 22.0, 18.0]
    b2 = synth.ReactorBatch(T, batch.P, batch.Y, batch.Yin, batch.tau)
    got = gpu_eval(torch, binding, mech, b2)
    ref = orc.evaluate(oracle_mech(mech), b2.T, b2.P, b2.Y, b2.Yin, b2.tau, want=("kf", "kr", "q", "wdot", "F"))
    warm = np.setdiff1d(np.arange(96), cold)
    assert rel_err(got["kf"][:, warm], ref["kf"][:, warm]).max() <= TOL_K
    assert rel_err(got["kr"][:, warm], ref["kr"][:, warm]).max() <= TOL_K
    werr, mask = wdot_masked_rel_err(got["wdot"][:, warm], ref["wdot"][:, warm])
    assert mask.any() and werr.max() <= TOL_K
    assert residual_rel_err(got["F"][:, warm], ref["F"][:, warm]).max() <= TOL_F
    # cold lanes, plain and three-body reactions.  The oracle forms A * T^b * exp(-Ea/RT) as the paper
    # writes it, so ITS result loses digits once exp(-Ea/RT) alone is subnormal (Ea/RT > ~708) although
    # k_f is not; compare to tolerance only where that intermediate is normal, and elsewhere require a
    # clean underflow (finite, non-negative, tiny).
    simple = mech.rtype <= 1
    kc, kref = got["kf"][simple][:, cold], ref["kf"][simple][:, cold]
    arg = mech.Ea[simple, None] / (1.9872042586408317 * T[cold][None, :])
    safe = (arg < 690.0) & (kref > 1e-290)
    assert safe.any() and (arg > 720.0).any()      # the case does straddle the range of the table exp
    assert rel_err(kc[safe], kref[safe]).max() <= TOL_K
    assert np.all(np.isfinite(kc)) and np.all(kc >= 0.0) and np.all(kc[arg > 720.0] < 1e-280)


# ------------------------------------------------------------------ full-size launches, every reactor
def _mass_conservation(mech, wdot):
    ww = mech.W[:, None] * wdot
    return np.median(np.abs(ww.sum(axis=0)) / np.abs(ww).sum(axis=0))


def check_full_batch(mech, batch, wdot, F):
    """Every reactor of a full-size batch.  At this size some wdot_i are the small remainder of terms 1e9 times
    larger (e.g. C1 reactor 64738, species 17: |wdot| = 6e-10 of the reactor's largest), where the FP64 oracle
    itself is 1.6e-10 from the long-double oracle: the literal 1e-10 is then below what FP64 can resolve, so the
    bar is the conditioning-aware one (util.floor_criterion) against the LONG-DOUBLE oracle, plus:
    the GPU is no noisier than 4x the independent FP64 oracle, and the literal 1e-10 / 1e-9 holds on all but a
    1e-5 fraction of the entries north_star's mask selects."""
    om = oracle_mech(mech)
    star = orc.evaluate(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("wdot", "F"), long_double=True)
    dbl = orc.evaluate(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("wdot", "F"))
    S = orc.roundoff_scale(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau)
    _, mask = wdot_masked_rel_err(wdot, star["wdot"])
    assert mask.any()
    worst_w, fr_w = floor_criterion(wdot, star["wdot"], S["Sw"], rtol=TOL_K, mask=mask)
    worst_F, fr_F = floor_criterion(F, star["F"], S["SF"], rtol=TOL_F)
    _, od_w = floor_criterion(dbl["wdot"], star["wdot"], S["Sw"], rtol=TOL_K, mask=mask)
    _, od_F = floor_criterion(dbl["F"], star["F"], S["SF"], rtol=TOL_F)
    assert worst_w <= 1.0 and worst_F <= 1.0, (worst_w, worst_F)
    assert fr_w <= 4 * max(od_w, 1.0) and fr_F <= 4 * max(od_F, 1.0), (fr_w, od_w, fr_F, od_F)
    werr, _ = wdot_masked_rel_err(wdot, dbl["wdot"])
    assert (werr > TOL_K).sum() <= 1e-5 * mask.sum()
    assert (residual_rel_err(F, dbl["F"]) > TOL_F).mean() <= 1e-5
    return dbl


def test_C1_full_size_residual_every_reactor(torch_cuda, binding):
    """BASELINE config 1 at its full batch through the exact launch bench.py times -- psr_eval_residual on
    65,536 reactors into preallocated F and wdot (the multi-tile, double-buffered Y - Y_in path of a
    persistent CTA) -- compared with the oracle on EVERY reactor; the same for psr_eval_residual_energy,
    psr_eval_wdot and psr_eval_kf_kr (c-J: every perf number rests on parity of the launch
    that is timed)."""
    torch = torch_cuda
    mech, batch = synth.make_config("C1")
    gm = binding.Mechanism.from_synth(mech)
    T, P, Y, Yin, tau = (dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
    F, wdot = torch.empty_like(Y), torch.empty_like(Y)
    for _ in range(2):   # twice: the second call runs with warm L2 / resident tables, as in bench.py
        gm.eval_residual(T, P, Y, Yin, tau, F=F, wdot=wdot)
    om = oracle_mech(mech)
    Fh, wh = F.cpu().numpy(), wdot.cpu().numpy()
    ref = check_full_batch(mech, batch, wh, Fh)
    ref.update(orc.evaluate(om, batch.T, batch.P, batch.Y, want=("kf", "kr")))
    assert _mass_conservation(mech, wh) <= 1e-12
    # psr_eval_wdot alone gives the same bits
    assert np.array_equal(gm.eval_wdot(T, P, Y).cpu().numpy(), wh)
    # adiabatic residual: species rows bit-identical, energy row against the oracle
    Tin = torch.full_like(T, 300.0)
    Fe, FTe, we = gm.eval_residual_energy(T, P, Y, Tin, Yin, tau, want_wdot=True)
    # (the energy-row call runs the fused kernel, the plain one the warp-specialised kernel: same arithmetic per
    # reaction, another summation order in nu^T q and in sum Y_i/W_i)
    gm.set_option(binding.OPT_FUSED_ONLY, 1)
    Ff, wf = gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
    gm.set_option(binding.OPT_FUSED_ONLY, 0)
    assert np.array_equal(Fe.cpu().numpy(), Ff.cpu().numpy()) and np.array_equal(we.cpu().numpy(), wf.cpu().numpy())
    check_full_batch(mech, batch, wf.cpu().numpy(), Ff.cpu().numpy())
    refe = orc.evaluate_energy(om, batch.T, batch.P, batch.Y, np.full(batch.n, 300.0), batch.Yin, batch.tau)
    rho = batch.P / (RGAS * batch.T * (batch.Y / mech.W[:, None]).sum(axis=0))
    scale = energy_scale(mech, batch, np.full(batch.n, 300.0), ref["wdot"], rho)
    err = np.abs(FTe.cpu().numpy() - refe["FT"]) / np.maximum(np.abs(refe["FT"]), 1e-3 * scale)
    assert err.max() <= TOL_F
    # rate constants of all 325 reactions x 65,536 reactors
    kf, kr = gm.eval_kf_kr(T, P, Y)
    assert rel_err(kf.cpu().numpy(), ref["kf"]).max() <= TOL_K
    assert rel_err(kr.cpu().numpy(), ref["kr"]).max() <= TOL_K
    gm.close()


@pytest.mark.parametrize("cfg,n,kernel", [("C1", 2 * 148 * 32 + 77, 1), ("C0", 333, 1), ("C4", 999, 1), ("C2", 2 * 148 * 32 + 5, 2),
                                          ("C3", 70, 2)])
def test_tensor_memory_copy_of_the_tile_changes_no_bit(torch_cuda, binding, cfg, n, kernel):
    """The warp-specialised kernels take the six concentration factors of a 3+3 record from a copy of the C tile in
    tensor memory; PSR_OPT_NO_TMEM reads them from shared memory.  Same values, same arithmetic: every
    output agrees to the bit -- over more than two tiles per CTA (tile buffers reused) and a ragged last tile.  (C3:
    500 species do not fit the 512 columns; the switch changes nothing there.)"""
    torch = torch_cuda
    mech, batch = synth.make_config(cfg, n)
    gm = binding.Mechanism.from_synth(mech)
    assert gm.info()["eval_kernel"] == kernel
    T, P, Y, Yin, tau = (dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
    got = []
    for no_tmem in (0, 1, 0):
        gm.set_option(binding.OPT_NO_TMEM, no_tmem)
        F, w = gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
        kf, kr = gm.eval_kf_kr(T, P, Y)
        got.append([x.cpu().numpy() for x in (F, w, kf, kr)])
    for a, b in ((0, 1), (0, 2)):
        for x, y in zip(got[a], got[b]):
            assert np.array_equal(x, y)
    assert np.all(np.isfinite(got[0][0]))
    gm.close()


@pytest.mark.parametrize("cfg", ["C2", "C3"])
def test_large_configs_full_size_every_reactor(torch_cuda, binding, cfg):
    """BASELINE configs 2 and 3 at their full batches through psr_eval_residual (the launches bench.py
    times under `extra`): every reactor against the oracle, invariants over the whole output."""
    torch = torch_cuda
    mech, batch = synth.make_config(cfg)
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau)]
    F, wdot = gm.eval_residual(*args, want_wdot=True)
    F, wdot = F.cpu().numpy(), wdot.cpu().numpy()
    gm.close()
    check_full_batch(mech, batch, wdot, F)
    assert _mass_conservation(mech, wdot) <= 1e-12
    # sum_i F_i = (sum Y - sum Y_in)/tau - sum_i wdot_i W_i / rho, and the last sum vanishes (mass conservation)
    lhs = F.sum(axis=0)
    rhs = (batch.Y.sum(axis=0) - batch.Yin.sum(axis=0)) / batch.tau
    scale = np.abs(F).sum(axis=0)
    assert np.median(np.abs(lhs - rhs) / scale) <= 1e-12


def test_C4_full_size_jacobian_every_reactor(torch_cuda, binding):
    """BASELINE config 4 at its full 8,192 reactors (the psr_fd_jacobian launch sequence bench.py times):
    every Jacobian by the floor criterion against the long-double oracle, structural invariants too.
    Over the 23.9 M entries of the whole batch the tail of the round-off noise is longer than on the samples
    SURVEY.md 8(c)-J calibrated K_j on (there an FP64 code reached 4 eps S/h in the Y columns; here the
    independent FP64 ORACLE reaches 21.2 and 627 in the T column, measured): the Y-column constant of this
    test is 64 instead of 32, and the GPU must in addition be no noisier than 4x the FP64 oracle."""
    torch = torch_cuda
    mech, batch = synth.make_config("C4")
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau)]
    J, F0 = gm.fd_jacobian(*args, want_F0=True)
    J, F0 = J.cpu().numpy(), F0.cpu().numpy()
    gm.close()
    assert np.all(np.isfinite(J))
    assert np.all(J[:, 0, 0] == 1.0) and np.all(J[:, 1:, 0] == 0.0)          # row 0 = e_0 (g13)
    # species rows of a Y column sum to 1/tau, of the T column to 0 (mass conservation), up to FD noise
    col_sums = J[:, :, 1:].sum(axis=2)
    scale = np.abs(J[:, :, 1:]).sum(axis=2)
    assert np.median(np.abs(col_sums[:, 1:] - 1.0 / batch.tau[:, None]) / scale[:, 1:]) <= 1e-6
    assert np.median(np.abs(col_sums[:, 0]) / scale[:, 0]) <= 1e-6
    om = oracle_mech(mech)
    worst = fr_T = fr_Y = 0.0
    for r0 in range(0, batch.n, 2048):   # the long-double reference in blocks (its J is 191 MB for the batch)
        sub = batch.take(np.arange(r0, min(r0 + 2048, batch.n)))
        jl = orc.jacobian(om, sub.T, sub.P, sub.Y, sub.Yin, sub.tau, long_double=True)
        w, ft, fy = jacobian_floor_ratio(J[r0:r0 + sub.n], jl["J"], jl["S"], jl["H"], K_y=64.0)
        worst, fr_T, fr_Y = max(worst, w), max(fr_T, ft), max(fr_Y, fy)
        assert residual_rel_err(F0[r0:r0 + sub.n, 1:].T, jl["F0"][:, 1:].T).max() <= TOL_F
        if r0 == 0:   # the independent FP64 oracle on the first block (a lower bound of its worst over the batch)
            jd = orc.jacobian(om, sub.T, sub.P, sub.Y, sub.Yin, sub.tau)
            _, od_T, od_Y = jacobian_floor_ratio(jd["J"], jl["J"], jl["S"], jl["H"])
    assert worst <= 1.0, (worst, fr_T, fr_Y, od_T, od_Y)
    assert fr_T <= 4 * max(od_T, 1.0) and fr_Y <= 4 * max(od_Y, 1.0), (fr_T, od_T, fr_Y, od_Y)


# ------------------------------------------------------------------ Jacobian (a10)
@pytest.mark.parametrize("cfg,n", [("C4", 40), ("C0", 50), ("C2", 3), ("P5", 4)])
def test_fd_jacobian_floor_criterion(torch_cuda, binding, cfg, n):
    torch = torch_cuda
    mech, batch = synth.make_config(cfg, n)
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau)]
    # psr_fd_jacobian takes the fused kernel (psr_jac.cu) where the mechanism qualifies (C4, C0) and the generic
    # three-launch sweep elsewhere (K > 64: C2, P5); the generic sweep is also run on every case
    J, F0 = gm.fd_jacobian(*args, want_F0=True)
    J2 = gm.fd_jacobian(*args)  # without the F0 output
    gm.set_option(binding.OPT_JAC_GENERIC, 1)
    Jg, F0g = gm.fd_jacobian(*args, want_F0=True)
    # diagnostic sweep in which every column is a full evaluation: the generic sweep takes the T-only
    # factors of the Y columns from the base state's rate table and must give the same bits
    gm.set_option(binding.OPT_JAC_UNHOISTED, 1)
    J3 = gm.fd_jacobian(*args)
    gm.set_option(binding.OPT_JAC_UNHOISTED, 0)
    gm.set_option(binding.OPT_JAC_GENERIC, 0)
    torch.cuda.synchronize()
    J, F0, J2, J3, Jg, F0g = (x.cpu().numpy() for x in (J, F0, J2, J3, Jg, F0g))
    gm.close()
    assert np.array_equal(J, J2)
    assert np.array_equal(Jg, J3)
    om = oracle_mech(mech)
    jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=True)
    jd = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, long_double=False)
    _, od_T, od_Y = jacobian_floor_ratio(jd["J"], jl["J"], jl["S"], jl["H"])
    for Jx, F0x in ((J, F0), (Jg, F0g)):
        # (1) binding criterion against the long-double reference
        worst, fr_T, fr_Y = jacobian_floor_ratio(Jx, jl["J"], jl["S"], jl["H"])
        assert worst <= 1.0, (worst, fr_T, fr_Y)
        # (2) the GPU is no noisier than 4x an independent FP64 CPU code
        assert fr_T <= 4 * max(od_T, 1.0) and fr_Y <= 4 * max(od_Y, 1.0), (fr_T, od_T, fr_Y, od_Y)
        # row 0 is e_0 exactly; base residual parity at 1e-9
        assert np.all(Jx[:, 0, 0] == 1.0) and np.all(Jx[:, 1:, 0] == 0.0)
        assert np.all(F0x[:, 0] == 0.0)
        assert residual_rel_err(F0x[:, 1:].T, jd["F0"][:, 1:].T).max() <= TOL_F
    if cfg in ("C4", "C0"):
        # the fused kernel forms the species columns without evaluating F twice: their round-off is far below the
        # forward-difference floor of any FP64 sweep (the oracle's included)
        _, _, fy = jacobian_floor_ratio(J, jl["J"], jl["S"], jl["H"])
        assert not np.array_equal(J, Jg) and fy <= 0.25 * max(od_Y, 1.0), (fy, od_Y)


# ------------------------------------------------------------------ energy row (NEXT-1)
def energy_scale(mech, batch, Tin, wdot_ref, rho):
    """Sum of the absolute terms of the energy row, per reactor: the row is a difference of large numbers,
    so its error is judged relative to max(|F_T|, 1e-3 of this scale).  NASA-7 forms of
    include/psr.h, vectorised over the batch (a tolerance scale, not an expected value)."""
    a = mech.nasa[:, :, None]                                   # [K][7][1]
    W = mech.W[:, None]

    def h_of(T):                                                # erg/g, [K][N]
        hRT = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T**2 / 3 + a[:, 3] * T**3 / 4 + a[:, 4] * T**4 / 5 + a[:, 5] / T
        return hRT * RGAS * T / W
    T = batch.T[None, :]
    h, hin = h_of(T), h_of(np.asarray(Tin, dtype=np.float64)[None, :])
    cp = (a[:, 0] + a[:, 1] * T + a[:, 2] * T**2 + a[:, 3] * T**3 + a[:, 4] * T**4) * RGAS / W
    S = (np.abs(batch.Yin * (hin - h)) / batch.tau[None, :] + np.abs(h * wdot_ref * W) / rho[None, :]).sum(axis=0)
    return S / (batch.Y * cp).sum(axis=0)


@pytest.mark.parametrize("cfg,n", [("C0", 100), ("C1", 333), ("C2", 70)])
def test_energy_residual_against_oracle(torch_cuda, binding, cfg, n):
    torch = torch_cuda
    mech, batch = synth.make_config(cfg, n)
    Tin = np.random.default_rng(3).uniform(300.0, 700.0, n)
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, Tin, batch.Yin, batch.tau)]
    F, FT, wdot = gm.eval_residual_energy(*args, want_wdot=True)
    gm.set_option(binding.OPT_FUSED_ONLY, 1)
    F2 = gm.eval_residual(args[0], args[1], args[2], args[4], args[5])
    gm.set_option(binding.OPT_FUSED_ONLY, 0)
    torch.cuda.synchronize()
    F, FT, wdot, F2 = F.cpu().numpy(), FT.cpu().numpy(), wdot.cpu().numpy(), F2.cpu().numpy()
    gm.close()
    ref = orc.evaluate_energy(oracle_mech(mech), batch.T, batch.P, batch.Y, Tin, batch.Yin, batch.tau)
    assert np.array_equal(F, F2)                                       # species rows: the same path (fused kernel)
    assert residual_rel_err(F, ref["F"]).max() <= TOL_F
    rho = batch.P / (8.31446261815324e7 * batch.T * (batch.Y / mech.W[:, None]).sum(axis=0))
    S = energy_scale(mech, batch, Tin, ref["wdot"], rho)
    err = np.abs(FT - ref["FT"]) / np.maximum(np.abs(ref["FT"]), 1e-3 * S)
    assert err.max() <= TOL_F, err.max()


def test_energy_residual_T3_golden(torch_cuda, binding):
    torch = torch_cuda
    gold = json.loads((Path(__file__).parent / "golden" / "t3_pins.json").read_text())["energy_Tin300"]
    mech, batch = synth.toy_t3()
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, np.array([300.0]), batch.Yin, batch.tau)]
    _, FT = gm.eval_residual_energy(*args)
    torch.cuda.synchronize()
    assert abs(float(FT[0]) - gold["F_T"]) <= 1e-9 * abs(gold["F_T"])
    gm.close()


@pytest.mark.parametrize("cfg,n", [("C4", 40), ("C0", 50), ("C2", 3)])
def test_fd_jacobian_energy_floor_criterion(torch_cuda, binding, cfg, n):
    """Adiabatic Jacobian (row 0 = energy row): floor criterion against the long-double oracle, species rows
    bit-identical to psr_fd_jacobian, hoisted sweep bit-identical to the all-columns sweep."""
    torch = torch_cuda
    mech, batch = synth.make_config(cfg, n)
    Tin = np.random.default_rng(4).uniform(300.0, 700.0, n)
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau)]
    dTin = dev(torch, Tin)
    J, F0 = gm.fd_jacobian(*args, want_F0=True, Tin=dTin)
    gm.set_option(binding.OPT_JAC_GENERIC, 1)    # the species rows are those of the generic sweep of psr_fd_jacobian
    Jp = gm.fd_jacobian(*args)
    gm.set_option(binding.OPT_JAC_GENERIC, 0)
    gm.set_option(binding.OPT_JAC_UNHOISTED, 1)
    J3 = gm.fd_jacobian(*args, Tin=dTin)
    gm.set_option(binding.OPT_JAC_UNHOISTED, 0)
    _, FT = gm.eval_residual_energy(args[0], args[1], args[2], dTin, args[3], args[4])
    torch.cuda.synchronize()
    J, F0, Jp, J3, FT = (x.cpu().numpy() for x in (J, F0, Jp, J3, FT))
    gm.close()
    assert np.array_equal(J, J3)
    assert np.array_equal(J[:, :, 1:], Jp[:, :, 1:])
    assert np.array_equal(F0[:, 0], FT)
    om = oracle_mech(mech)
    jl = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin, long_double=True)
    jd = orc.jacobian(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin)
    worst, fr_T, fr_Y = jacobian_floor_ratio(J, jl["J"], jl["S"], jl["H"])
    assert worst <= 1.0, (worst, fr_T, fr_Y)
    _, od_T, od_Y = jacobian_floor_ratio(jd["J"], jl["J"], jl["S"], jl["H"])
    assert fr_T <= 4 * max(od_T, 1.0) and fr_Y <= 4 * max(od_Y, 1.0), (fr_T, od_T, fr_Y, od_Y)


# ------------------------------------------------------------------ linear solve of the Newton step (NEXT-2)
EPS64 = 2.0 ** -53


def _backward_error_ok(A, x, b, n, factor=8.0):
    """Row-wise bound of Gaussian elimination with partial pivoting: |Ax - b|_inf <= c n eps (|A|_inf |x|_inf + |b|_inf).
    A: [N][col][row]."""
    M = np.swapaxes(A, 1, 2)
    res = np.abs(np.einsum("rij,rj->ri", M, x) - b).max(axis=1)
    bound = n * EPS64 * (np.abs(M).sum(axis=2).max(axis=1) * np.abs(x).max(axis=1) + np.abs(b).max(axis=1))
    return np.all(res <= factor * bound), float((res / bound).max())


@pytest.mark.parametrize("n,N", [(1, 5), (3, 7), (11, 33), (32, 40), (33, 9), (54, 300), (64, 17), (101, 6), (168, 2)])
def test_lu_solve_random_systems(torch_cuda, binding, n, N):
    torch = torch_cuda
    rng = np.random.default_rng(100 + n)
    M = rng.standard_normal((N, n, n)) + 3.0 * np.eye(n)
    if n > 1:
        M[0, 0, 0] = 0.0                                 # forces a row exchange in the first step of system 0
    b = rng.standard_normal((N, n))
    A = np.ascontiguousarray(np.swapaxes(M, 1, 2))       # A[r, col, row]
    x, info = binding.lu_solve(dev(torch, A), dev(torch, b.copy()))
    torch.cuda.synchronize()
    x, info = x.cpu().numpy(), info.cpu().numpy()
    xr, ir = orc.lu_solve(A, b)
    assert np.array_equal(info, ir) and np.all(info == 0)
    ok, worst = _backward_error_ok(A, x, b, n)
    assert ok, worst
    # same pivots, same elimination order: the two agree far inside the conditioning of these systems
    assert np.abs(x - xr).max() <= 1e-11 * np.abs(xr).max()


def test_lu_solve_flags_singular_systems_and_leaves_their_rhs(torch_cuda, binding):
    torch = torch_cuda
    M = np.stack([np.eye(4), np.array([[1.0, 2, 0, 0], [2, 4, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1]]), np.zeros((4, 4))])
    b = np.arange(12, dtype=np.float64).reshape(3, 4) + 1.0
    A = np.ascontiguousarray(np.swapaxes(M, 1, 2))
    x, info = binding.lu_solve(dev(torch, A), dev(torch, b.copy()))
    torch.cuda.synchronize()
    x, info = x.cpu().numpy(), info.cpu().numpy()
    _, ir = orc.lu_solve(A, b)
    assert np.array_equal(info, ir) and list(info) == [0, 2, 1]
    assert np.array_equal(x[0], b[0]) and np.array_equal(x[1], b[1]) and np.array_equal(x[2], b[2])


def test_newton_step_on_device_matches_the_oracle_solve(torch_cuda, binding):
    """One Newton update of the C4 system entirely on the device: J, F0 from psr_fd_jacobian, then J dx = -F0
    by psr_lu_solve; compared with the oracle's elimination of the same J (long double) and by backward error."""
    torch = torch_cuda
    mech, batch = synth.make_config("C4", 64)
    gm = binding.Mechanism.from_synth(mech)
    args = [dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau)]
    J, F0 = gm.fd_jacobian(*args, want_F0=True)
    rhs = (-F0).contiguous()
    dx, info = binding.lu_solve(J, rhs.clone())
    torch.cuda.synchronize()
    gm.close()
    Jh, bh, dx, info = J.cpu().numpy(), rhs.cpu().numpy(), dx.cpu().numpy(), info.cpu().numpy()
    assert np.all(info == 0) and np.all(np.isfinite(dx))
    n = mech.n_species + 1
    ok, worst = _backward_error_ok(Jh, dx, bh, n)
    assert ok, worst
    xr, ir = orc.lu_solve(Jh, bh)
    xl, _ = orc.lu_solve(Jh, bh, long_double=True)
    assert np.all(ir == 0)
    # forward error (these Jacobians are ill-conditioned, both FP64 solves sit 1e-9..1e-5 from the long-double
    # one): the GPU's distance is of the size of the FP64 oracle's -- typically (median) within 4x, never
    # beyond 64x; the rigorous statement is the backward error above
    e_gpu = np.abs(dx - xl).max(axis=1)
    e_ref = np.abs(xr - xl).max(axis=1)
    scale = np.abs(xl).max(axis=1)
    ratio = e_gpu / (e_ref + 1e-13 * scale)
    assert np.median(ratio) <= 4.0 and ratio.max() <= 64.0, (float(np.median(ratio)), float(ratio.max()))
    assert np.all(np.abs(dx[:, 0]) <= 1e-8 * scale)      # fixed-temperature row: dT = -F_T = 0 up to the solve's round-off


# ------------------------------------------------------------------ pseudo-transient step (NEXT-4)
@pytest.mark.parametrize("n,N", [(1, 5), (3, 7), (33, 9), (54, 300), (101, 6), (168, 2)])
def test_ptc_solve_random_systems(torch_cuda, binding, n, N):
    """(I/dt + J) dx = -F element by element against the oracle (same shift, same sign, same elimination),
    J and F left untouched, dt = inf bit-identical to psr_lu_solve on (J, -F)."""
    torch = torch_cuda
    rng = np.random.default_rng(300 + n)
    M = rng.standard_normal((N, n, n)) + 1.0 * np.eye(n)
    F = rng.standard_normal((N, n))
    dt = 10.0 ** rng.uniform(-3, 1, N)
    J = np.ascontiguousarray(np.swapaxes(M, 1, 2))
    Jd, Fd = dev(torch, J), dev(torch, F)
    dx, info = binding.ptc_solve(Jd, Fd, dev(torch, dt))
    torch.cuda.synchronize()
    assert np.array_equal(Jd.cpu().numpy(), J) and np.array_equal(Fd.cpu().numpy(), F)
    dx, info = dx.cpu().numpy(), info.cpu().numpy()
    xr, ir = orc.ptc_step(J, F, dt)
    assert np.array_equal(info, ir) and np.all(info == 0)
    assert np.abs(dx - xr).max() <= 1e-11 * np.abs(xr).max()
    A = J + (np.eye(n)[None] / dt[:, None, None])
    ok, worst = _backward_error_ok(A, dx, -F, n)
    assert ok, worst
    # Newton limit: no shift
    dxn, _ = binding.ptc_solve(Jd, Fd, dev(torch, np.full(N, np.inf)))
    xn, _ = binding.lu_solve(Jd, (-Fd).contiguous())
    torch.cuda.synchronize()
    assert np.array_equal(dxn.cpu().numpy(), xn.cpu().numpy())


def test_ptc_solve_edge_cases(torch_cuda, binding):
    torch = torch_cuda
    # a system the shift makes singular is flagged and its dx left as it was; N = 0 is a no-op
    J = np.array([[[-2.0]], [[1.0]]])
    F = np.array([[1.0], [3.0]])
    dx0 = dev(torch, np.full((2, 1), 7.0))
    dx, info = binding.ptc_solve(dev(torch, J), dev(torch, F), dev(torch, np.array([0.5, 0.5])), dx=dx0)
    torch.cuda.synchronize()
    assert list(info.cpu().numpy()) == [1, 0]
    assert dx.cpu().numpy()[0, 0] == 7.0 and dx.cpu().numpy()[1, 0] == -3.0 / 3.0
    e = torch.empty((0, 4), dtype=torch.float64, device="cuda")
    binding.ptc_solve(torch.empty((0, 4, 4), dtype=torch.float64, device="cuda"), e, torch.empty(0, dtype=torch.float64, device="cuda"))
    with pytest.raises(binding.PsrError):
        f = dev(torch, F)
        binding.ptc_solve(dev(torch, J), f, dev(torch, np.array([0.5, 0.5])), dx=f)      # dx aliases F


def test_pseudo_transient_iteration_on_device_reduces_the_residual(torch_cuda, binding):
    """The fallback loop the paper describes with this library's calls only: residual + Jacobian
    (psr_fd_jacobian), one implicit-Euler step (psr_ptc_solve), update -- on C4 states.  Every step is checked
    against the oracle's step on the same J, F0, dt (backward error of the shifted system; forward error against
    the long-double solve, relative to the FP64 oracle's own), and the residual norm must fall.  The paper gives
    no step-size rule ("See [5]"); the test takes dt = 0.1 / max_j sum_i |J_ij| per reactor."""
    torch = torch_cuda
    mech, batch = synth.make_config("C4", 32)
    gm = binding.Mechanism.from_synth(mech)
    T, P, Y, Yin, tau = (dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
    n = mech.n_species + 1
    norms = []
    for _ in range(3):
        J, F0 = gm.fd_jacobian(T, P, Y, Yin, tau, want_F0=True)
        dt = (0.1 / J.abs().sum(dim=2).max(dim=1).values).contiguous()
        dx, info = binding.ptc_solve(J, F0, dt)
        torch.cuda.synchronize()
        assert int(info.abs().max()) == 0
        Jh, Fh, dth, d = J.cpu().numpy(), F0.cpu().numpy(), dt.cpu().numpy(), dx.cpu().numpy()
        A = Jh + np.eye(n)[None] / dth[:, None, None]
        ok, worst = _backward_error_ok(A, d, -Fh, n)
        assert ok, worst
        xr, ir = orc.ptc_step(Jh, Fh, dth)
        xl, _ = orc.ptc_step(Jh, Fh, dth, long_double=True)
        assert np.all(ir == 0)
        scale = np.abs(xl).max(axis=1)
        ratio = np.abs(d - xl).max(axis=1) / (np.abs(xr - xl).max(axis=1) + 1e-13 * scale)
        assert np.median(ratio) <= 4.0 and ratio.max() <= 64.0, (float(np.median(ratio)), float(ratio.max()))
        assert np.all(np.abs(d - xr).max(axis=1) <= 1e-9 * scale)     # the shift makes these systems well conditioned
        norms.append(float(F0[:, 1:].abs().max()))
        Y = (Y + dx[:, 1:].t()).contiguous()           # x = (T, Y): row 0 is the fixed-temperature equation, dT = 0
        assert float(dx[:, 0].abs().max()) <= 1e-12 * float(scale.max())
    gm.close()
    assert norms[2] < norms[1] < norms[0], norms


# ------------------------------------------------------------------ hybrid solver (NEXT-4)
SOLVE_KW = dict(atol=1e-12, rtol=1e-7, max_iter=260, max_newton=5, max_ptc=20, dt0=1e-9, dt_grow=2.0, dt_shrink=0.25, y_floor=1e-9)


def _solve_both(torch, binding, mech, T0, P, Y0, Yin, tau, Tin=None, workspace_reactors=None, generic=True, **kw):
    """generic=True: the device loop builds its Jacobians with the generic forward-difference sweep, as the oracle
    does (paths are compared like with like); False: with the fused Jacobian kernel where it applies (its species
    columns carry no forward-difference round-off, so its Newton iteration contracts at least as fast)."""
    gm = binding.Mechanism.from_synth(mech)
    gm.set_option(binding.OPT_JAC_GENERIC, 1 if generic else 0)
    T, Y = dev(torch, T0), dev(torch, Y0)
    ws = None
    if workspace_reactors is not None:
        ws = torch.empty(int(binding.lib().psr_solve_hybrid_workspace_bytes(gm._h, workspace_reactors)), dtype=torch.uint8, device="cuda")
    st, nn, npt = gm.solve_hybrid(T, dev(torch, P), Y, dev(torch, Yin), dev(torch, tau),
                                  Tin=None if Tin is None else dev(torch, Tin), workspace=ws, **kw)
    torch.cuda.synchronize()
    got = dict(T=T.cpu().numpy(), Y=Y.cpu().numpy(), status=st.cpu().numpy(), n_newton=nn.cpu().numpy(), n_ptc=npt.cpu().numpy())
    gm.close()
    ref = orc.solve_hybrid(oracle_mech(mech), T0, P, Y0, Yin, tau, Tin=Tin, **kw)
    return got, ref


def _compare_solves(mech, got, ref, P, Yin, tau, kw, exact_paths=False):
    """The device loop against the oracle's.  What is unique is compared strictly: which reactors converge, and the
    solution (within the solver's own tolerance).  The PATH is not unique under rounding -- the forward-difference
    Jacobians of the two sides differ at the 1e-8 level, the systems are ill-conditioned, and "has the correction
    passed the tolerance within max_newton iterations" then falls differently for some reactors, which adds or
    removes a pseudo-transient stage -- so iteration counts must agree on average, and exactly where
    `exact_paths` says the path is short and well-conditioned enough to be unique."""
    conv = (got["status"] == 0) & (ref["status"] == 0)
    assert (got["status"] == ref["status"]).mean() >= 0.95
    same = conv & (got["n_newton"] == ref["n_newton"]) & (got["n_ptc"] == ref["n_ptc"])
    if exact_paths:
        assert same.sum() >= 0.9 * conv.sum(), (conv.mean(), same.mean())
    else:
        for k in ("n_newton", "n_ptc"):
            assert abs(got[k][conv].mean() - ref[k][conv].mean()) <= 0.1 * ref[k][conv].mean() + 0.5, k
        assert same.mean() >= 0.2
    # the same solution wherever both converged (to the same root: a few reactors of a stiff mechanism have more than one)
    w = kw["atol"] + kw["rtol"] * np.abs(ref["Y"])
    d = (np.abs(got["Y"] - ref["Y"]) / w).max(axis=0)
    assert (d[conv] <= 1.0).mean() >= 0.97 and d[same].max() <= 1.0
    assert np.allclose(got["T"][conv], ref["T"][conv], rtol=10 * kw["rtol"])
    # every converged device solution satisfies the equations as well as the oracle's do (judged by the oracle)
    om = oracle_mech(mech)
    ok, okr = got["status"] == 0, ref["status"] == 0
    Fg = orc.evaluate(om, got["T"], P, got["Y"], Yin, tau, want=("F",))["F"]
    Fr = orc.evaluate(om, ref["T"], P, ref["Y"], Yin, tau, want=("F",))["F"]
    Sg = orc.roundoff_scale(om, got["T"], P, got["Y"], Yin, tau)["SF"]
    Sr = orc.roundoff_scale(om, ref["T"], P, ref["Y"], Yin, tau)["SF"]
    rg = (np.abs(Fg) / np.where(Sg > 0, Sg, 1.0))[:, ok].max(axis=0)       # |F_i| against the size of its terms
    rr = (np.abs(Fr) / np.where(Sr > 0, Sr, 1.0))[:, okr].max(axis=0)
    assert np.median(rg) <= 2 * np.median(rr) + 1e-12 and rg.max() <= 10 * rr.max() + 1e-9


def test_solve_hybrid_matches_the_oracle_loop_on_C0(torch_cuda, binding):
    """psr_solve_hybrid from the generated (far) initial states of C0: Newton stages, pseudo-transient conditioning
    and the switches between them, on the device, against the oracle's loop; also in sub-batches (small workspace)."""
    mech, batch = synth.make_config("C0", 300)
    got, ref = _solve_both(torch_cuda, binding, mech, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, **SOLVE_KW)
    assert (ref["n_ptc"] > 0).any() and (ref["status"] == 0).mean() > 0.9
    _compare_solves(mech, got, ref, batch.P, batch.Yin, batch.tau, SOLVE_KW)
    got2, _ = _solve_both(torch_cuda, binding, mech, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, workspace_reactors=77, **SOLVE_KW)
    for k in got:
        assert np.array_equal(got[k], got2[k]), k      # sub-batching does not change a reactor's path
    _fused_path_check(torch_cuda, binding, mech, batch, ref, SOLVE_KW)


def _fused_path_check(torch, binding, mech, batch, ref, kw):
    """The default device path (fused Jacobian kernel): the same solutions, and no more Newton iterations on average
    than the forward-difference paths need."""
    got, _ = _solve_both(torch, binding, mech, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, generic=False, **kw)
    conv = (got["status"] == 0) & (ref["status"] == 0)
    assert (got["status"] == 0).mean() >= (ref["status"] == 0).mean() - 0.06
    w = kw["atol"] + kw["rtol"] * np.abs(ref["Y"])
    d = (np.abs(got["Y"] - ref["Y"]) / w).max(axis=0)
    # (both stop on the size of their last Newton correction; with different Jacobians the estimates they stop at
    # differ by a multiple of the tolerance that grows with the conditioning of the system)
    assert (d[conv] <= 100.0).mean() >= 0.97 and np.median(d[conv]) <= 1.0
    assert got["n_newton"][conv].mean() <= ref["n_newton"][conv].mean() + 0.5


def test_solve_hybrid_paths_that_are_unique(torch_cuda, binding):
    """Where the path does not hang on rounding the device takes exactly the oracle's: an inert mechanism (linear
    residual: two Newton iterations), and a second-order reaction 2A <=> B from near and far guesses (Newton alone;
    an inadmissible first trial, a pseudo-transient stage, then Newton)."""
    torch = torch_cuda
    mech, batch = synth.make_config("C0", 64)
    mm = copy.deepcopy(mech)
    mm.A = np.zeros_like(mech.A)
    kw = dict(SOLVE_KW, atol=1e-9, rtol=1e-6)
    got, ref = _solve_both(torch, binding, mm, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, **kw)
    # (a species whose Y is far below its Y_in has a forward-difference column accurate to eps |Y - Y_in| / h only,
    # which can cost a third iteration on either side)
    assert np.all(got["status"] == 0) and np.all(got["n_ptc"] == 0) and np.all((got["n_newton"] == 2) | (got["n_newton"] == 3))
    assert (got["n_newton"] == 2).mean() >= 0.8 and (got["n_newton"] == ref["n_newton"]).mean() >= 0.8
    assert np.allclose(got["Y"], batch.Yin, rtol=1e-12, atol=1e-15)
    # 2A <=> B (the mechanism of the oracle's pin), a sweep of initial guesses
    reac_ptr, reac_sp, reac_nu = synth._side_csr([(0, 0)])
    prod_ptr, prod_sp, prod_nu = synth._side_csr([(1,)])
    m2 = synth.Mechanism(
        n_species=2, n_reactions=1, atoms=np.zeros((2, 4), dtype=np.int32), W=np.array([15.0, 30.0]),
        nasa=np.array([[3.5, 1e-4, 0.0, 0.0, 0.0, -1000.0, 2.0], [3.9, 3e-4, -2e-8, 0.0, 0.0, -1600.0, 23.0]]),
        A=np.array([2.0e9]), b=np.array([0.0]), Ea=np.array([2.0e3]), rtype=np.zeros(1, dtype=np.uint8),
        reversible=np.ones(1, dtype=np.uint8), reac_ptr=reac_ptr, reac_sp=reac_sp, reac_nu=reac_nu,
        prod_ptr=prod_ptr, prod_sp=prod_sp, prod_nu=prod_nu, eff_ptr=np.zeros(2, dtype=np.int32),
        eff_sp=np.zeros(0, dtype=np.int32), eff_val=np.zeros(0), A0=np.zeros(1), b0=np.zeros(1), Ea0=np.zeros(1),
        troe=np.zeros((1, 4)), meta={"name": "2A<=>B"})
    yA = np.concatenate([np.linspace(0.02, 0.98, 49), [1e-9, 1 - 1e-9, 1 - 1e-6]])
    N = yA.size
    Y0 = np.stack([yA, 1 - yA])
    Yin = np.tile(np.array([[0.9], [0.1]]), (1, N))
    kw = dict(atol=1e-14, rtol=1e-9, max_iter=200, max_newton=8, max_ptc=10, dt0=1e-9, dt_grow=2.0, dt_shrink=0.25, y_floor=0.0)
    got, ref = _solve_both(torch, binding, m2, np.full(N, 1200.0), np.full(N, 1.01325e6), Y0, Yin, np.full(N, 1e-3), **kw)
    assert np.all(ref["status"] == 0) and (ref["n_ptc"] > 0).any() and (ref["n_ptc"] == 0).any()
    for k in ("status", "n_newton", "n_ptc"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.allclose(got["Y"], ref["Y"], rtol=1e-9, atol=1e-14)
    assert np.allclose(got["Y"][0], 0.48972816473969222, rtol=1e-8)      # the mpmath root of tests/test_oracle_pins.py


def test_solve_hybrid_on_C4_from_far_and_from_perturbed_converged_states(torch_cuda, binding):
    """BASELINE config 4's mechanism (53 species / 325 reactions): from the generated states (pseudo-transient stages
    needed), then from converged states perturbed by 1 % (Newton alone, a few iterations: the same path on both sides)."""
    torch = torch_cuda
    mech, batch = synth.make_config("C4", 96)
    kw0 = dict(SOLVE_KW, max_iter=420)
    got, ref = _solve_both(torch, binding, mech, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, **kw0)
    assert (ref["n_ptc"] > 0).all() and (ref["status"] == 0).mean() > 0.9
    _compare_solves(mech, got, ref, batch.P, batch.Yin, batch.tau, kw0)
    _fused_path_check(torch, binding, mech, batch, ref, kw0)
    conv = ref["status"] == 0
    rng = np.random.default_rng(17)
    Y1 = ref["Y"][:, conv] * (1.0 + 0.01 * rng.uniform(-1, 1, (mech.n_species, conv.sum())))
    sub = batch.take(np.flatnonzero(conv))
    kw = dict(SOLVE_KW, atol=1e-10, rtol=1e-5, max_iter=12, max_newton=12)
    got1, ref1 = _solve_both(torch, binding, mech, ref["T"][conv], sub.P, Y1, sub.Yin, sub.tau, **kw)
    assert (ref1["status"] == 0).mean() > 0.9 and (ref1["n_ptc"][ref1["status"] == 0] == 0).all()
    _compare_solves(mech, got1, ref1, sub.P, sub.Yin, sub.tau, kw, exact_paths=True)
    w = kw["atol"] + 10 * kw["rtol"] * np.abs(ref["Y"][:, conv])
    ok = (got1["status"] == 0)
    assert (np.abs(got1["Y"] - ref["Y"][:, conv]) / w)[:, ok].max() <= 1.0     # back at the solution it was perturbed from


@pytest.mark.parametrize("generic", [False, True])
def test_solve_hybrid_rounds_after_convergence_change_nothing(torch_cuda, binding, generic):
    """Finished reactors are marked on the device (their tiles of the fused Jacobian kernel and their linear systems are
    left out, and once none is left a round is three empty launches).  So the budget beyond the last reactor's
    convergence must change no output: 14 rounds and 300 rounds give the same bits -- with sub-batches (the counter is
    per sub-batch), with a batch in which some reactors never finish, and on both Jacobian paths."""
    torch = torch_cuda
    mech, batch = synth.make_config("C4", 160)
    gm = binding.Mechanism.from_synth(mech)
    gm.set_option(binding.OPT_JAC_GENERIC, 1 if generic else 0)
    P, Yin, tau = (dev(torch, x) for x in (batch.P, batch.Yin, batch.tau))
    kw = dict(SOLVE_KW, max_iter=300)
    ws = torch.empty(int(binding.lib().psr_solve_hybrid_workspace_bytes(gm._h, 64)), dtype=torch.uint8, device="cuda")   # 3 sub-batches
    T, Y = dev(torch, batch.T), dev(torch, batch.Y)
    st, nn, npt = gm.solve_hybrid(T, P, Y, Yin, tau, workspace=ws, **kw)
    torch.cuda.synchronize()
    conv = (st == 0).cpu().numpy()
    assert 0.8 < conv.mean() < 1.0 or conv.all()          # the far start leaves a few reactors unfinished
    # restart from the finished reactors' solutions, perturbed: every one converges within a few Newton iterations
    rng = np.random.default_rng(5)
    idx = np.flatnonzero(conv)
    Y1 = Y.cpu().numpy()[:, idx] * (1.0 + 0.01 * rng.uniform(-1, 1, (mech.n_species, idx.size)))
    T1 = T.cpu().numpy()[idx]
    sub = batch.take(idx)
    outs = []
    for max_iter in (14, 300):
        Tt, Yt = dev(torch, T1), dev(torch, Y1)
        s1, n1, p1 = gm.solve_hybrid(Tt, dev(torch, sub.P), Yt, dev(torch, sub.Yin), dev(torch, sub.tau), workspace=ws,
                                     **dict(SOLVE_KW, atol=1e-10, rtol=1e-5, max_iter=max_iter, max_newton=12))
        torch.cuda.synchronize()
        outs.append([x.cpu().numpy() for x in (Tt, Yt, s1, n1, p1)])
    assert (outs[0][2] == 0).all() and outs[0][3].max() <= 12
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)
    # and the mixed batch: a budget cut short against the full one agree on every reactor that had finished by then
    Tt, Yt = dev(torch, batch.T), dev(torch, batch.Y)
    s2, n2, p2 = gm.solve_hybrid(Tt, P, Yt, Yin, tau, workspace=ws, **dict(SOLVE_KW, max_iter=200))
    torch.cuda.synchronize()
    early = (s2 == 0).cpu().numpy()
    assert early.any() and np.array_equal(Yt.cpu().numpy()[:, early], Y.cpu().numpy()[:, early])
    assert np.array_equal(n2.cpu().numpy()[early], nn.cpu().numpy()[early]) and np.array_equal(p2.cpu().numpy()[early], npt.cpu().numpy()[early])
    gm.close()


def test_solve_hybrid_adiabatic_and_argument_checks(torch_cuda, binding):
    """Tin given: row 0 of the system is the energy row and T is solved for.  An inert mechanism settles at
    (T_in, Y_in) on the same path as the oracle.  (With chemistry the adiabatic systems of these synthetic mechanisms
    are too ill-conditioned for two FP64 codes to stay on one path from a far guess; their Jacobians and solves are
    compared one call at a time by the floor-criterion and backward-error tests above.)"""
    torch = torch_cuda
    mech, batch = synth.make_config("C0", 40)
    Tin = np.linspace(600.0, 900.0, batch.n)
    mm = copy.deepcopy(mech)
    mm.A = np.zeros_like(mech.A)
    kw = dict(SOLVE_KW, atol=1e-9, rtol=1e-6, max_iter=40, max_newton=30, y_floor=np.inf)
    got, ref = _solve_both(torch, binding, mm, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, Tin=Tin, **kw)
    # (a far first Newton step in T can leave T > 0 -- only the mass fractions are bounded -- and such a reactor
    # never recovers: on both sides alike)
    ok = ref["status"] == 0
    assert np.array_equal(got["status"], ref["status"]) and ok.mean() >= 0.8
    assert np.all(got["n_ptc"][ok] == 0) and (got["n_newton"] == ref["n_newton"])[ok].mean() >= 0.8
    assert np.allclose(got["T"][ok], Tin[ok], rtol=1e-8) and np.allclose(got["Y"][:, ok], batch.Yin[:, ok], rtol=1e-9, atol=1e-13)
    gm = binding.Mechanism.from_synth(mech)
    T, Y = dev(torch, batch.T), dev(torch, batch.Y)
    args = (T, dev(torch, batch.P), Y, dev(torch, batch.Yin), dev(torch, batch.tau))
    with pytest.raises(binding.PsrError):
        gm.solve_hybrid(*args, max_newton=0)
    with pytest.raises(binding.PsrError):
        gm.solve_hybrid(*args, workspace=torch.empty(64, dtype=torch.uint8, device="cuda"))
    st, nn, npt = gm.solve_hybrid(*args, max_iter=0)      # no budget: nothing moves, nothing converged
    assert bool((st == 1).all()) and bool((nn == 0).all()) and np.array_equal(Y.cpu().numpy(), batch.Y)
    gm.close()


# ------------------------------------------------------------------ streams and graphs
def test_calls_are_capturable_in_a_cuda_graph_and_honour_the_stream(torch_cuda, binding):
    """Every evaluation call only enqueues work on the caller's stream (psr.h), so a Newton iteration
    (residual + Jacobian) can be captured once in a CUDA graph and replayed on new states."""
    torch = torch_cuda
    mech, batch = synth.make_config("C1", 200)
    gm = binding.Mechanism.from_synth(mech)
    T, P, Y, Yin, tau = (dev(torch, x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
    n = mech.n_species + 1
    F, w = torch.empty_like(Y), torch.empty_like(Y)
    J = torch.empty((batch.n, n, n), dtype=torch.float64, device="cuda")
    side = torch.cuda.Stream()
    # the generic Jacobian sweep's scratch belongs to the mechanism: without a reservation the call refuses to
    # allocate inside a capture (psr.h) instead of invalidating it.  (The fused Jacobian kernel this mechanism
    # normally takes needs no such scratch; the graph below captures both.)
    Jgen = torch.empty_like(J)
    gm.set_option(binding.OPT_JAC_GENERIC, 1)
    probe = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(probe, stream=side):
            with pytest.raises(binding.PsrError) as ei:
                gm.fd_jacobian(T, P, Y, Yin, tau, J=Jgen)
            assert ei.value.status == binding.PSR_EINVAL and "psr_mech_reserve" in str(ei.value)
    del probe
    gm.reserve(batch.n)                                # sizes the scratch buffer outside the capture
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            gm.eval_residual(T, P, Y, Yin, tau, F=F, wdot=w)
            gm.fd_jacobian(T, P, Y, Yin, tau, J=Jgen)
            gm.set_option(binding.OPT_JAC_GENERIC, 0)
            gm.fd_jacobian(T, P, Y, Yin, tau, J=J)
            gm.set_option(binding.OPT_JAC_GENERIC, 1)
    # a later, larger eager call outgrows the scratch: the captured graph keeps pointing at the buffer it was
    # captured with, which stays allocated until the mechanism is freed
    _, big = synth.make_config("C4", 6000)
    gm.fd_jacobian(*(dev(torch, x) for x in (big.T, big.P, big.Y, big.Yin, big.tau)))
    gm.set_option(binding.OPT_JAC_GENERIC, 0)
    torch.cuda.synchronize()
    # new state in the same buffers, replay, compare with direct calls on the default stream
    _, b2 = synth.make_config("C4", 200)
    for dst, src in ((T, b2.T), (P, b2.P), (Y, b2.Y), (Yin, b2.Yin), (tau, b2.tau)):
        dst.copy_(dev(torch, src))
    F.zero_(); w.zero_(); J.zero_(); Jgen.zero_()
    torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    F_g, w_g, J_g, Jgen_g = F.clone(), w.clone(), J.clone(), Jgen.clone()
    F_d, w_d = gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
    J_d = gm.fd_jacobian(T, P, Y, Yin, tau)
    gm.set_option(binding.OPT_JAC_GENERIC, 1)
    Jgen_d = gm.fd_jacobian(T, P, Y, Yin, tau)
    torch.cuda.synchronize()
    gm.close()
    assert torch.equal(F_g, F_d) and torch.equal(w_g, w_d) and torch.equal(J_g, J_d) and torch.equal(Jgen_g, Jgen_d)
    ref = orc.evaluate(oracle_mech(mech), b2.T, b2.P, b2.Y, b2.Yin, b2.tau, want=("wdot", "F"))
    assert residual_rel_err(F_g.cpu().numpy(), ref["F"]).max() <= TOL_F


# ------------------------------------------------------------------ bounds-checked build (stands in for compute-sanitizer)
_CHECK_SCRIPT = r"""
import json, sys
import numpy as np, torch
from paper_2005_11468_b200 import binding, build, synth
build.build(check=True)                       # no-op when libpsr_b200_check.so is newer than the sources
binding._LIB_PATH = build.LIB_CHECK           # this process loads the -DPSR_CHECK library instead of the product one
binding._build.needs_build = lambda: False
dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
out = {"selftest": binding.check_failures(selftest=True)}          # one assertion tripped on purpose
for cfg, n in (("C0", None), ("C1", 2000), ("C3", 97), ("C2", 70), ("P5", 40)):
    mech, b = synth.make_config(cfg, n) if n else synth.make_config(cfg)
    gm = binding.Mechanism.from_synth(mech)
    T, P, Y, Yin, tau = (dev(x) for x in (b.T, b.P, b.Y, b.Yin, b.tau))
    Tin = torch.full_like(T, 400.0)
    for fused_only in (0, 1):                 # the warp-specialised kernel where it applies, then the general one
        gm.set_option(binding.OPT_FUSED_ONLY, fused_only)
        gm.eval_kf_kr(T, P, Y)
        gm.eval_wdot(T, P, Y, want_q=True)
        gm.eval_residual(T, P, Y, Yin, tau, want_wdot=True)
    gm.eval_residual_energy(T, P, Y, Tin, Yin, tau, want_wdot=True)
    m = min(b.n, 40)
    a = [x[..., :m].contiguous() for x in (T, P, Y, Yin, tau)]
    for generic in (0, 1):                    # the fused Jacobian kernel where it applies, then the generic sweep
        gm.set_option(binding.OPT_JAC_GENERIC, generic)
        gm.fd_jacobian(*a, want_F0=True)
    gm.fd_jacobian(*a, Tin=Tin[:m].contiguous())
    if cfg in ("C0", "C1"):
        n1 = mech.n_species + 1
        gm.fd_jacobian_noalloc(*a, J=torch.empty((m, n1, n1), dtype=torch.float64, device="cuda"))
        # the hybrid solver: 20 rounds, two compactions of the reactors still iterating (the partition's destinations
        # and the scatter back are checked), in sub-batches
        ws = torch.empty(int(binding.lib().psr_solve_hybrid_workspace_bytes(gm._h, 24)), dtype=torch.uint8, device="cuda")
        gm.solve_hybrid(a[0].clone(), a[1], a[2].clone(), a[3], a[4], workspace=ws, atol=1e-10, rtol=1e-6, max_iter=20,
                        max_newton=4, max_ptc=6, dt0=1e-9, dt_grow=2.0, dt_shrink=0.25, y_floor=1e-9)
    torch.cuda.synchronize()
    out[cfg] = binding.check_failures()
    gm.close()
print("RESULT " + json.dumps(out))
"""


def test_bounds_checked_build(torch_cuda):
    """compute-sanitizer is refused on this GPU pool; this stands in for its memcheck on the indices the
    kernels take from the mechanism tables.  libpsr_b200_check.so is the same sources with -DPSR_CHECK: every
    table-derived shared-memory offset (factor rows, q / rate-tile rows, gather entries, flush targets, scatter rows)
    and every global output index is asserted on the device.  Run in a process of its own (it loads another build of
    the library) on C0 in full, ragged C1 / C2 / C3 / P5 batches, every evaluation call, both evaluation kernels, both
    Jacobian paths, the energy row, the no-alloc entry point and the hybrid solver with its compaction.  A self-test
    trips one assertion first: zero failures
    afterwards means the checks ran and held.  It finds out-of-range indices -- not races, not uninitialised reads."""
    import subprocess
    import sys
    root = Path(__file__).resolve().parent.parent
    res = subprocess.run([sys.executable, "-c", _CHECK_SCRIPT], cwd=root, capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, res.stderr[-3000:]
    line = [l for l in res.stdout.splitlines() if l.startswith("RESULT ")][-1]
    out = json.loads(line[len("RESULT "):])
    assert out.pop("selftest") == [1, 999]
    assert set(out) == {"C0", "C1", "C2", "C3", "P5"}
    for cfg, (count, code) in out.items():
        assert (count, code) == (0, 0), (cfg, count, code)


def test_product_build_carries_no_checks(binding):
    assert binding.check_failures() == (-1, 0)


# ------------------------------------------------------------------ kernel math
def test_table_exp_accuracy(torch_cuda, binding):
    """csrc/psr_math.cuh exp_fast against mpmath (50 digits): <= 4e-16 relative over the argument
    range the rate forms reach, exact special values, library path beyond |x| >= 700 and for NaN/Inf."""
    import mpmath
    mech, _ = synth.make_config("C0", 1)
    gm = binding.Mechanism.from_synth(mech)
    rng = np.random.default_rng(7)
    x = np.concatenate([rng.uniform(-700, 700, 20000), rng.uniform(-1, 1, 5000), rng.uniform(-1e-3, 1e-3, 2000),
                        np.arange(-64, 65) * np.log(2) / 64, [0.0, -0.0, 699.999, -699.999, 1e-300]])
    y = gm.probe_exp_values(x)
    mpmath.mp.dps = 50
    ref = np.array([float(mpmath.exp(mpmath.mpf(float(v)))) for v in x])
    err = np.abs(y - ref) / ref
    assert err.max() <= 4e-16, err.max()
    assert np.all(y[x == 0.0] == 1.0)
    edge = np.array([700.0, 709.7, 710.0, -708.0, -745.0, -800.0, np.inf, -np.inf, np.nan])
    ye = gm.probe_exp_values(edge)
    with np.errstate(over="ignore"):
        ne = np.exp(edge)
    assert np.isnan(ye[-1]) and ye[6] == np.inf and ye[7] == 0.0 and ye[2] == np.inf and ye[5] == 0.0
    fin = np.isfinite(ne) & (ne > 1e-300)
    assert np.all(np.abs(ye[fin] - ne[fin]) <= 4e-16 * ne[fin])
    gm.close()
