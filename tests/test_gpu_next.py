"""Parity of the NEXT rows of SURVEY.md 8(f) on the GPU (`-m gpu`): quasi-eigenstates (NEXT-3, tbpm_propagate_qe), the Haydock
recursion (NEXT-2, tbpm_haydock) and the AC-conductivity correlation (NEXT-4, tbpm_corr_ac) against the oracle's plain statements (oracle.quasi_eigenstates / oracle.haydock, themselves
pinned in tests/test_oracle_next_pins.py), element by element on the same seeded inputs."""
import math

import numpy as np
import pytest
import torch

from paper_2509_26309_b200 import tbpm, workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def to_np(w):
    return (w.hop_i.cpu().numpy(), w.hop_j.cpu().numpy(), w.hop_val.cpu().numpy(),
            None if w.onsite is None else w.onsite.cpu().numpy())


@pytest.mark.parametrize("cfg,over,n_state,n_step", [
    (2, dict(Na=48, Nb=40), 3, 24),                                  # padded tile of 4, diagonal
    (3, dict(Na=64, Nb=48), 1, 16),                                  # irregular rows, single state
    (4, dict(Lx=128, Ly=24, phi_den=32), 8, 12),                     # complex hops, rolling-window kernel
    (5, dict(L=32), 11, 9),                                          # lattice kernel tile + padded tile of 4
])
def test_quasi_eigenstates(dev, oracle_mod, cfg, over, n_state, n_step):
    w = W.make_workload(cfg, device=dev, **over)
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    energies = [0.0, 0.31 * w.rescale, -0.77 * w.rescale]
    corr, norm2, qe = tbpm.tbpm_propagate_qe(H, psi0, energies, n_step, w.dt, w.rescale)
    ref_c, _, _ = tbpm.tbpm_propagate(H, psi0, n_step, w.dt, w.rescale)
    assert (corr - ref_c).abs().max() <= 1e-13                       # the same propagation (small models: another kernel, rounding only)
    hi, hj, hv, on = to_np(w)
    ref = oracle_mod.quasi_eigenstates(w.n_orb, on, hi, hj, hv, psi0.cpu().numpy(), energies, n_step, w.dt, w.rescale)
    assert qe.shape == (n_state, 3, w.n_orb)
    scale = np.abs(ref).max()
    assert np.abs(qe.cpu().numpy() - ref).max() <= 1e-10 * max(1.0, scale)
    assert np.abs(norm2.cpu().numpy() - 1).max() <= 1e-12


def test_quasi_eigenstates_eigenstate_closed_form_and_edges(dev):
    """psi0 an eigenstate (uniform state of the clean cubic lattice, E0 = 6t): qe[e] = psi0 * sum_n w_n exp(i (E_e - E0) n dt)."""
    L, s, n_step = 32, 15.0, 20
    n, hi, hj, hv = W.cubic_hops(L, -1.0, dev)
    H = tbpm.tbpm_build(n, None, hi, hj, hv)
    psi0 = torch.full((8, n), 1 / math.sqrt(n), dtype=torch.complex128, device=dev)
    dt = math.pi / s
    energies = [-6.0, -5.0, 3.3]
    _, _, qe = tbpm.tbpm_propagate_qe(H, psi0, energies, n_step, dt, s)
    k = np.arange(n_step + 1)
    wn = 0.5 * (1 + np.cos(np.pi * k / n_step))
    for e, Ee in enumerate(energies):
        g = (wn * np.exp(1j * (Ee + 6.0) * k * dt)).sum()
        assert np.abs(qe[:, e].cpu().numpy() - g / math.sqrt(n)).max() <= 1e-10
    with pytest.raises(tbpm.TbpmError):                              # more than 16 energies
        tbpm.tbpm_propagate_qe(H, psi0, list(range(17)), 2, dt, s)
    c, _, q0 = tbpm.tbpm_propagate_qe(H, psi0, [], 3, dt, s)         # no energies: plain propagation
    assert q0.shape == (8, 0, n) and c.shape == (8, 3)


@pytest.mark.parametrize("cfg,over,n_site,n_iter", [
    (2, dict(Na=48, Nb=40), 5, 40),                                  # honeycomb + disorder, padded tile of 8
    (3, dict(Na=64, Nb=48), 3, 32),                                  # vacancies
    (4, dict(Lx=128, Ly=96, phi_den=32), 8, 24),                     # complex hops (Landau levels: the recursion loses orthogonality early)
    (5, dict(L=32), 12, 64),                                         # cubic + strong disorder: lattice kernel, two tiles
])
def test_haydock_coefficients(dev, oracle_mod, cfg, over, n_site, n_iter):
    """a_n, b_n of the first n_iter <= 64 levels to 1e-10 (relative to the spectral scale) against the oracle's recursion.
    (The map (H, site) -> (a_n, b_n) is ill-conditioned once Ritz values converge -- any two floating-point Lanczos runs part
    company there -- so the cases stop before that: the wave front has not wrapped round the sample.)"""
    w = W.make_workload(cfg, device=dev, **over)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    sites = W.ldos_sites(w.n_orb, n_site)
    a, b = tbpm.tbpm_haydock(H, sites, n_iter)
    hi, hj, hv, on = to_np(w)
    ra, rb = oracle_mod.haydock(w.n_orb, on, hi, hj, hv, sites.numpy(), n_iter)
    assert (rb > 0).all()
    assert np.abs(a.cpu().numpy() - ra).max() <= 1e-10 * w.rescale
    assert np.abs(b.cpu().numpy() - rb).max() <= 1e-10 * w.rescale


def test_haydock_chain_closed_form_and_ldos(dev, oracle_mod):
    """Ring of N sites: a_n = eps, b_1 = sqrt(2)|t|, b_n = |t|; and the LDOS from the GPU coefficients equals the exact
    Green function of a small disordered model (continued fraction, oracle.haydock_ldos)."""
    N, t = 4096, -1.3
    i = torch.arange(N, dtype=torch.int32, device=dev)
    H = tbpm.tbpm_build(N, torch.full((N,), 0.7, dtype=torch.float64, device=dev), i, ((i + 1) % N).to(torch.int32),
                        torch.full((N,), t, dtype=torch.complex128, device=dev))
    a, b = tbpm.tbpm_haydock(H, [17, 2000], 50)
    a, b = a.cpu().numpy(), b.cpu().numpy()
    assert np.abs(a - 0.7).max() <= 1e-12
    assert np.abs(b[:, 0] - math.sqrt(2) * abs(t)).max() <= 1e-12 and np.abs(b[:, 1:] - abs(t)).max() <= 1e-12
    w = W.make_workload(5, device=dev, L=4)                          # N = 64
    Hs = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    a, b = tbpm.tbpm_haydock(Hs, [11], 80)
    hi, hj, hv, on = to_np(w)
    Hd = np.zeros((64, 64), dtype=np.complex128)
    Hd[hi, hj] = hv
    Hd[hj, hi] = np.conj(hv)
    Hd[np.arange(64), np.arange(64)] += on
    Ej, V = np.linalg.eigh(Hd)
    E = np.linspace(-w.rescale, w.rescale, 201)
    exact = -(np.abs(V[11]) ** 2 / (E[:, None] + 0.4j - Ej[None, :])).sum(axis=1).imag / np.pi
    got = oracle_mod.haydock_ldos(a[0].cpu().numpy(), b[0].cpu().numpy(), E, 0.4)
    assert np.abs(got - exact).max() <= 1e-9 * exact.max()
    dev_ldos = tbpm.tbpm_haydock_ldos(a, b, torch.as_tensor(E, device=dev), 0.4)      # the continued fraction on the device
    assert np.abs(dev_ldos[0].cpu().numpy() - got).max() <= 1e-12 * exact.max()
    assert tbpm.lib().tbpm_haydock(Hs.handle, None, 0, 5, None, None, None, 0, None) == tbpm.TBPM_OK   # n_site = 0
    with pytest.raises(tbpm.TbpmError):
        tbpm.tbpm_haydock(Hs, [64], 3)


@pytest.mark.parametrize("Lx,Ly,phi_den,n_state,n_step,beta,mu,axes", [
    (64, 24, 16, 3, 10, 2.0, 0.4, (0, 1)),                           # padded tile of 4; sigma_xy-type correlation
    (128, 16, 32, 8, 6, 6.0, -0.8, (0, 0)),                          # W = 128: H runs on the square-lattice kernel; sigma_xx
    (48, 40, 8, 9, 5, 1.0, 0.0, (1, 1)),                             # tile of 8 + padded tile of 1; sigma_yy
])
def test_corr_ac(dev, oracle_mod, Lx, Ly, phi_den, n_state, n_step, beta, mu, axes):
    """NEXT-4: <psi2(t)|J_a|psi1(t)> with psi1 = [1 - f(H)] J_b psi0, psi2 = f(H) psi0, every entry against the oracle."""
    w = W.make_workload(4, device=dev, Lx=Lx, Ly=Ly, phi_den=phi_den)
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    J, jn = [], []
    for ax in axes:
        n, ji, jj, jv = W.square_current_hops(Lx, Ly, ax, phi_den=phi_den, device=dev)
        J.append(tbpm.tbpm_build(n, None, ji, jj, jv))
        jn.append((ji.cpu().numpy(), jj.cpu().numpy(), jv.cpu().numpy()))
    corr = tbpm.tbpm_corr_ac(H, J[0], J[1], psi0, n_step, w.dt, w.rescale, beta, mu)
    hi, hj, hv, on = to_np(w)
    ref = oracle_mod.corr_ac(w.n_orb, on, hi, hj, hv, jn[0], jn[1], psi0.cpu().numpy(), n_step, w.dt, w.rescale, beta, mu)
    assert corr.shape == (n_state, n_step + 1)
    assert np.abs(corr.cpu().numpy() - ref).max() <= 1e-10 * max(1.0, np.abs(ref).max())
    again = tbpm.tbpm_corr_ac(H, J[0], J[1], psi0, n_step, w.dt, w.rescale, beta, mu)
    assert torch.equal(corr, again)                                  # deterministic


@pytest.mark.parametrize("L,n_state,n_step,beta,mu", [(32, 8, 5, 0.4, 1.0), (12, 3, 7, 1.5, -2.0)])
def test_corr_dp(dev, oracle_mod, L, n_state, n_step, beta, mu):
    """NEXT-4, dynamic polarisation: <psi2(t)| rho(q) |psi1(t)> with psi1 = [1 - f(H)] rho(-q) psi0 on the disordered cubic lattice
    (L = 32: H runs on the three-dimensional lattice kernel), every entry against the oracle."""
    w = W.make_workload(5, device=dev, L=L)
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    idx = torch.arange(w.n_orb, device=dev)
    ph = (2 * math.pi / L) * (1.0 * (idx % L) + 2.0 * (idx // (L * L))).to(torch.float64)
    rho = torch.complex(torch.cos(ph), torch.sin(ph))
    corr = tbpm.tbpm_corr_dp(H, rho, rho.conj().contiguous(), psi0, n_step, w.dt, w.rescale, beta, mu)
    hi, hj, hv, on = to_np(w)
    ref = oracle_mod.corr_dp(w.n_orb, on, hi, hj, hv, rho.cpu().numpy(), rho.conj().cpu().numpy(), psi0.cpu().numpy(), n_step, w.dt,
                             w.rescale, beta, mu)
    assert np.abs(corr.cpu().numpy() - ref).max() <= 1e-10 * max(1.0, np.abs(ref).max())
