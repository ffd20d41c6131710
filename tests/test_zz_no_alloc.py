"""tbpm_propagate_static: the propagation with the library's static device array as workspace (no allocation inside the call).

Collected last on purpose (the suite runs with `pytest -x`).  The new entry point is compared with the existing path
(`tbpm_propagate` with a caller workspace) on two calls in a row that share the static array: the second call has fewer states and
another model size, so it runs over the first call's left-overs.  Same kernels, same launch configuration, same order of the
reductions: the results must agree bit for bit, and both must agree with the oracle within the tolerance of the parity tests.
"""
import numpy as np
import pytest
import torch

from paper_2509_26309_b200 import tbpm, workloads as W

pytestmark = pytest.mark.gpu

CORR_TOL = 1e-10     # north_star, as in tests/test_gpu_parity.py
NORM_TOL = 1e-12


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def both_paths(dev, w, n_state, n_step):
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    assert tbpm.tbpm_propagate_bytes(H, n_state) <= tbpm.TBPM_STATIC_WORKSPACE_BYTES
    corr_ref, norm_ref, _ = tbpm.tbpm_propagate(H, psi0, n_step, w.dt, w.rescale)
    # outputs allocated by the caller beforehand and filled with garbage: the call must write every entry
    corr = torch.full((n_state, n_step), float("nan"), dtype=torch.complex128, device=dev)
    norm2 = torch.full((n_state, n_step), float("nan"), dtype=torch.float64, device=dev)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(dev)
    tbpm.tbpm_propagate_static(H, psi0, n_step, w.dt, w.rescale, corr=corr, norm2=norm2)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == before                # nothing went through torch's allocator either
    return H, psi0, corr_ref, norm_ref, corr, norm2


def check(corr_ref, norm_ref, corr, norm2):
    assert (corr - corr_ref).abs().max().item() <= CORR_TOL
    assert (norm2 - norm_ref).abs().max().item() <= NORM_TOL
    assert (norm2 - 1).abs().max().item() <= NORM_TOL
    assert torch.equal(corr.view(torch.float64), corr_ref.view(torch.float64))       # in fact bit-identical
    assert torch.equal(norm2, norm_ref)


def test_static_workspace_two_calls_in_a_row(dev, oracle_mod):
    # call 1: cubic 16^3 + Anderson disorder, 8 states (one tile of 8: the launch-per-term path, 4096 x 8 elements per vector)
    w1 = W.make_workload(5, device=dev, L=16)
    H1, psi1, cr1, nr1, c1, n1 = both_paths(dev, w1, 8, 6)
    check(cr1, nr1, c1, n1)
    # call 2, straight after, on the same array: BASELINE.json:configs[0] (honeycomb 64 x 64, one state: the one-launch cluster path)
    w2 = W.make_workload(1, device=dev)
    H2, psi2, cr2, nr2, c2, n2 = both_paths(dev, w2, 1, 16)
    check(cr2, nr2, c2, n2)
    # a square lattice with flux, 8 states: the two-terms-per-sweep kernel, its two extra vectors inside the static array too
    w4 = W.make_workload(4, device=dev, Lx=128, Ly=24, phi_den=32)
    H4, psi4, cr4, nr4, c4, n4 = both_paths(dev, w4, 8, 5)
    check(cr4, nr4, c4, n4)
    assert tbpm.tbpm_last_launch_count(H4) == 1 + 5 * 11             # 10 pairs + reduction per time step: the pair path ran
    # call 3: the first model again, three states (a padded tile of 4) over call 2's left-overs, against the oracle itself
    psi3 = w1.psi0(device=dev, n_state=3)
    c3, n3 = tbpm.tbpm_propagate_static(H1, psi3, 5, w1.dt, w1.rescale)
    ref, refn = oracle_mod.propagate(w1.n_orb, w1.onsite.cpu().numpy(), w1.hop_i.cpu().numpy(), w1.hop_j.cpu().numpy(),
                                     w1.hop_val.cpu().numpy(), psi3.cpu().numpy(), 5, w1.dt, w1.rescale)[:2]
    assert np.abs(c3.cpu().numpy() - ref).max() <= CORR_TOL
    assert np.abs(n3.cpu().numpy() - refn).max() <= NORM_TOL
    # repeated call: bit-identical (the array's previous contents do not leak into the result)
    c4, n4 = tbpm.tbpm_propagate_static(H1, psi3, 5, w1.dt, w1.rescale)
    assert torch.equal(c3.view(torch.float64), c4.view(torch.float64)) and torch.equal(n3, n4)


def test_static_workspace_limits(dev):
    w = W.make_workload(2, device=dev, Na=256, Nb=256)               # 131,072 orbitals x 4 states: 33.6 MB of vectors
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    assert tbpm.tbpm_propagate_bytes(H, 4) > tbpm.TBPM_STATIC_WORKSPACE_BYTES
    psi0 = w.psi0(device=dev, n_state=4)
    launches = tbpm.tbpm_total_launch_count()
    with pytest.raises(tbpm.TbpmError) as e:
        tbpm.tbpm_propagate_static(H, psi0, 2, w.dt, w.rescale)
    assert e.value.code == tbpm.TBPM_ETOOBIG and "TBPM_STATIC_WORKSPACE_BYTES" in str(e.value)
    assert tbpm.tbpm_total_launch_count() == launches               # rejected before anything was launched
    # empty calls succeed and touch nothing, as in tbpm_propagate
    c, n = tbpm.tbpm_propagate_static(H, psi0[:0], 3, w.dt, w.rescale)
    assert c.shape == (0, 3)
