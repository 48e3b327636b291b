"""psr_fd_jacobian_noalloc -- the entry point for callers that cannot let the library allocate (include/psr.h).

Same fused Jacobian kernel as psr_fd_jacobian, its scratch in a static device array of the library instead of the
buffer psr_mech_load allocates.  Checked against the existing path on two calls in a row with DIFFERENT states: the
array keeps the first call's contents, so anything the kernel read before rewriting it would show in the second.

This file is collected last on purpose (pytest -x: a failure here hides no other test); it passes
alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2005_11468_b200 import synth
from util import jacobian_floor_ratio, oracle_mech, residual_rel_err

pytestmark = pytest.mark.gpu

TOL_F = 1e-9          # residual / Jacobian tolerance of tests/test_gpu_parity.py (BASELINE.json: north_star)


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


def test_noalloc_jacobian_matches_the_existing_path_on_two_calls_in_a_row(torch_cuda, binding):
    torch = torch_cuda
    mech, big = synth.make_config("C4", 2 * 1111)
    n = mech.n_species + 1
    gm = binding.Mechanism.from_synth(mech)
    om = oracle_mech(mech)
    # two batches of 1,111 reactors (35 tiles, the last one ragged), different states
    batches = [big.take(np.arange(0, 1111)), big.take(np.arange(1111, 2222))]
    J = torch.empty((1111, n, n), dtype=torch.float64, device="cuda")
    F0 = torch.empty((1111, n), dtype=torch.float64, device="cuda")
    for call, b in enumerate(batches):
        args = [dev(torch, x) for x in (b.T, b.P, b.Y, b.Yin, b.tau)]
        J.fill_(float("nan"))
        F0.fill_(float("nan"))
        gm.fd_jacobian_noalloc(*args, J=J, F0=F0)                  # caller-owned outputs, nothing allocated inside
        J_ref, F0_ref = gm.fd_jacobian(*args, want_F0=True)        # the existing path
        torch.cuda.synchronize()
        Jn, Fn, Jr, Fr = J.cpu().numpy(), F0.cpu().numpy(), J_ref.cpu().numpy(), F0_ref.cpu().numpy()
        assert np.all(np.isfinite(Jn)) and np.all(np.isfinite(Fn)), call
        # the tolerance the parity tests use: 1e-9 on residual and Jacobian entries (relative; entries that are exactly
        # zero in one are exactly zero in the other: row 0 = e_0)
        assert residual_rel_err(Fn[:, 1:].T, Fr[:, 1:].T).max() <= TOL_F, call
        assert np.array_equal(Jn == 0.0, Jr == 0.0), call
        nz = Jr != 0.0
        assert (np.abs(Jn - Jr)[nz] / np.abs(Jr)[nz]).max() <= TOL_F, call
        # it is the same kernel on the same tiles: the two paths agree to the bit
        assert np.array_equal(Jn, Jr) and np.array_equal(Fn, Fr), call
        # and against the oracle, by the criterion of test_fd_jacobian_floor_criterion, on a sample
        idx = np.array([0, 1, 31, 32, 555, 1109, 1110])
        sub = b.take(idx)
        jl = orc.jacobian(om, sub.T, sub.P, sub.Y, sub.Yin, sub.tau, long_double=True)
        worst, fr_T, fr_Y = jacobian_floor_ratio(Jn[idx], jl["J"], jl["S"], jl["H"])
        assert worst <= 1.0, (call, worst, fr_T, fr_Y)
    # F0 may be left out
    args = [dev(torch, x) for x in (batches[0].T, batches[0].P, batches[0].Y, batches[0].Yin, batches[0].tau)]
    J2 = torch.empty_like(J)
    gm.fd_jacobian_noalloc(*args, J=J2)
    torch.cuda.synchronize()
    assert np.array_equal(J2.cpu().numpy(), gm.fd_jacobian(*args).cpu().numpy())
    gm.close()


def test_noalloc_jacobian_rejects_what_is_beyond_its_limits(torch_cuda, binding):
    """More reactions than the static scratch is sized for, and mechanisms the fused kernel does not take, are refused
    with a clear error and nothing is launched (the outputs keep their contents)."""
    torch = torch_cuda
    for cfg, needle in (("C3", "reactions"), ("C2", "does not qualify")):   # 2,500 reactions > 2,048; 200 species > 64
        mech, b = synth.make_config(cfg, 40)
        n = mech.n_species + 1
        gm = binding.Mechanism.from_synth(mech)
        args = [dev(torch, x) for x in (b.T, b.P, b.Y, b.Yin, b.tau)]
        J = torch.full((b.n, n, n), -7.0, dtype=torch.float64, device="cuda")
        with pytest.raises(binding.PsrError) as ei:
            gm.fd_jacobian_noalloc(*args, J=J)
        assert ei.value.status == binding.PSR_EUNSUPPORTED and needle in str(ei.value), str(ei.value)
        torch.cuda.synchronize()
        assert bool((J == -7.0).all())
        gm.close()
    # argument checks, N = 0
    mech, b = synth.make_config("C4", 8)
    gm = binding.Mechanism.from_synth(mech)
    lib = binding.lib()
    assert lib.psr_fd_jacobian_noalloc(gm._h, 4, None, None, None, None, None, 4, None, None, None) == binding.PSR_EINVAL
    assert lib.psr_fd_jacobian_noalloc(gm._h, 0, None, None, None, None, None, 0, None, None, None) == binding.PSR_OK
    gm.close()
