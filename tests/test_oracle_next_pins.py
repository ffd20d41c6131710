"""Pins of the oracle's NEXT rows -- quasi-eigenstates (NEXT-3) and the Haydock recursion (NEXT-2) -- against what the
mathematics fixes (all CPU, `-m "not gpu"`): exact diagonalisation (numpy.linalg.eigh), closed forms of the chain, the
moments <i|H^m|i> from dense matrix powers, and the route through the time-domain LDOS correlation.
"""
import math

import numpy as np
import pytest

from paper_2509_26309_b200 import workloads as W
from test_oracle_pins import dense_h, np_hops


def hann(n_step):
    return 0.5 * (1.0 + np.cos(np.pi * np.arange(n_step + 1) / n_step))


# ---- NEXT-3: quasi-eigenstates --------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,over", [
    (2, dict(Na=10, Nb=8)),                           # honeycomb + Anderson disorder
    (4, dict(Lx=12, Ly=10, phi_den=4)),               # complex hops
    (5, dict(L=6)),                                   # cubic + strong disorder
])
def test_qe_exact_diagonalisation(oracle_mod, cfg, over):
    """qe[e] = sum_j phi_j <phi_j|psi0> sum_n w_n exp(i (E_e - E_j) n dt): a wrong sign of the phase, a missing n = 0 term,
    a shifted window or an off-by-one in the time index each fail."""
    w = W.make_workload(cfg, **over)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=2).numpy()
    H = dense_h(w.n_orb, hi, hj, hv, on)
    Ej, V = np.linalg.eigh(H)
    n_step = 40
    energies = np.array([Ej[3], 0.37 * w.rescale, -0.81 * w.rescale])
    qe = oracle_mod.quasi_eigenstates(w.n_orb, on, hi, hj, hv, psi0, energies, n_step, w.dt, w.rescale)
    assert qe.shape == (2, 3, w.n_orb)
    n = np.arange(n_step + 1)
    wn = hann(n_step)
    for b in range(2):
        cj = V.conj().T @ psi0[b]
        for e, Ee in enumerate(energies):
            f = (wn[None, :] * np.exp(1j * np.outer(Ee - Ej, n) * w.dt)).sum(axis=1)      # [j]
            ref = V @ (cj * f)
            assert np.abs(qe[b, e] - ref).max() < 1e-12


def test_qe_eigenstate_closed_form(oracle_mod):
    """psi0 an eigenstate with energy E0 (uniform state of the clean honeycomb lattice, E0 = 3t): qe[e] = psi0 * g(E_e - E0)
    with g(d) = sum_n w_n exp(i d n dt); at E_e = E0 the sum is n_step / 2 + 1/2 exactly (Hann weights)."""
    w = W.make_workload(1, Na=12, Nb=12)
    hi, hj, hv, on = np_hops(w)
    psi0 = np.full((1, w.n_orb), 1 / math.sqrt(w.n_orb), dtype=np.complex128)
    E0 = 3 * -2.7
    n_step = 32
    energies = np.array([E0, E0 + 0.5, 2.0])
    qe = oracle_mod.quasi_eigenstates(w.n_orb, on, hi, hj, hv, psi0, energies, n_step, w.dt, w.rescale)
    n = np.arange(n_step + 1)
    for e, Ee in enumerate(energies):
        g = (hann(n_step) * np.exp(1j * (Ee - E0) * n * w.dt)).sum()
        assert np.abs(qe[0, e] - psi0[0] * g).max() < 1e-12
    assert abs((qe[0, 0] / psi0[0])[0] - (n_step / 2 + 0.5)) < 1e-12


# ---- NEXT-2: Haydock recursion --------------------------------------------------------------------------------------
def test_haydock_chain_closed_forms(oracle_mod):
    """Textbook coefficients: open chain from its END site: a_n = 0, b_n = |t| (semi-infinite chain); ring from any site:
    b_1 = sqrt(2)|t|, then |t| (until the two arms meet at N/2); on-site energy eps shifts every a_n by eps."""
    N, t = 200, -1.3
    i = np.arange(N - 1, dtype=np.int32)
    a, b = oracle_mod.haydock(N, None, i, i + 1, np.full(N - 1, t + 0j), [0], 40)
    assert np.abs(a).max() < 1e-14 and np.abs(b - abs(t)).max() < 1e-13
    i = np.arange(N, dtype=np.int32)
    eps = np.full(N, 0.7)
    a, b = oracle_mod.haydock(N, eps, i, ((i + 1) % N).astype(np.int32), np.full(N, t + 0j), [17], 40)
    assert np.abs(a - 0.7).max() < 1e-13
    assert abs(b[0, 0] - math.sqrt(2) * abs(t)) < 1e-13 and np.abs(b[0, 1:] - abs(t)).max() < 1e-13


@pytest.mark.parametrize("cfg,over", [
    (2, dict(Na=10, Nb=8)), (3, dict(Na=12, Nb=12)), (4, dict(Lx=12, Ly=10, phi_den=4)), (5, dict(L=6)),
])
def test_haydock_moments_and_krylov(oracle_mod, cfg, over):
    """The Jacobi matrix J of (a, b) reproduces the moments: (J^m)_00 = <i|H^m|i> for m <= 2 n_iter - 1 (dense matrix powers);
    a wrong sign, a missing b_n phi_{n-1} term or an index shift in b fails at low m.  Also: b > 0 and a real."""
    w = W.make_workload(cfg, **over)
    hi, hj, hv, on = np_hops(w)
    H = dense_h(w.n_orb, hi, hj, hv, on)
    n_iter = 7
    sites = W.ldos_sites(w.n_orb, 3).numpy()
    a, b = oracle_mod.haydock(w.n_orb, on, hi, hj, hv, sites, n_iter)
    for s, site in enumerate(sites):
        J = np.diag(a[s]) + np.diag(b[s, :-1], 1) + np.diag(b[s, :-1], -1)
        Hm = np.eye(w.n_orb, dtype=np.complex128)
        Jm = np.eye(n_iter)
        for m in range(1, 2 * n_iter):
            Hm = Hm @ H
            Jm = Jm @ J
            mu = Hm[site, site]
            assert abs(mu.imag) < 1e-9 * max(1.0, abs(mu))
            assert abs(Jm[0, 0] - mu.real) <= 1e-11 * max(1.0, abs(mu.real)), (m, Jm[0, 0], mu)
    assert (b > 0).all()


def test_haydock_ldos_matches_exact_green_function(oracle_mod):
    """With enough levels to exhaust the Krylov space of a small model (N = 64; 80 levels, the recursion simply goes on in
    floating point) the continued fraction IS G_ii(z) = sum_j |phi_j(i)|^2 / (z - E_j)."""
    w = W.make_workload(5, L=4)                                     # N = 64, strong disorder: no degeneracies
    hi, hj, hv, on = np_hops(w)
    H = dense_h(w.n_orb, hi, hj, hv, on)
    Ej, V = np.linalg.eigh(H)
    site = 11
    E = np.linspace(-w.rescale, w.rescale, 301)
    eta = 0.4
    exact = -(np.abs(V[site]) ** 2 / (E[:, None] + 1j * eta - Ej[None, :])).sum(axis=1).imag / np.pi
    a, b = oracle_mod.haydock(w.n_orb, on, hi, hj, hv, [site], 80)
    got = oracle_mod.haydock_ldos(a[0], b[0], E, eta)
    assert np.abs(got - exact).max() < 1e-10 * exact.max()


def test_haydock_agrees_with_time_domain_ldos(oracle_mod):
    """Second, independent route to the same quantity: the TBPM LDOS correlation <i|psi_i(t)> (oracle.ldos) windowed and
    transformed (oracle.dos_from_corr) against the Haydock continued fraction at a matching broadening."""
    w = W.make_workload(5, L=10)
    hi, hj, hv, on = np_hops(w)
    site = int(W.ldos_sites(w.n_orb, 1)[0])
    n_step = 64
    corr, _ = oracle_mod.ldos(w.n_orb, on, hi, hj, hv, [site], n_step, w.dt, w.rescale)
    E, D = oracle_mod.dos_from_corr(corr[0], w.rescale)
    a, b = oracle_mod.haydock(w.n_orb, on, hi, hj, hv, [site], 60)
    eta = 2.0 * w.rescale / n_step                                  # the Hann window's resolution
    Hd = oracle_mod.haydock_ldos(a[0], b[0], E, eta)
    assert abs(np.trapezoid(D, E) - 1.0) < 2e-2 and abs(np.trapezoid(Hd, E) - 1.0) < 6e-2
    # first and second moments of the two spectra agree (the broadening kernels differ, the low moments do not)
    m1d, m1h = np.trapezoid(E * D, E) / np.trapezoid(D, E), np.trapezoid(E * Hd, E) / np.trapezoid(Hd, E)
    assert abs(m1d - m1h) < 0.05 * w.rescale
    assert abs(m1d - on[site]) < 0.05 * w.rescale                   # <i|H|i> = onsite_i


# ---- NEXT-4: AC-conductivity correlation ----------------------------------------------------------------------------
@pytest.mark.parametrize("beta,mu,s", [(2.0, 0.3, 4.8), (11.0, -1.0, 4.8), (0.5, 0.0, 9.0)])
def test_fermi_chebyshev_closed_form(oracle_mod, beta, mu, s):
    """sum_k c_k T_k(x) = 1 / (exp(beta (s x - mu)) + 1) on [-1, 1]; the complement sums to 1 - f; |c_k| decays."""
    c = oracle_mod.fermi_cheb_coeff(beta, mu, s)
    g = oracle_mod.fermi_cheb_coeff(beta, mu, s, one_minus=True)
    x = np.linspace(-1, 1, 201)
    T = np.cos(np.outer(np.arange(c.size), np.arccos(x)))
    f = 1.0 / (np.exp(beta * (s * x - mu)) + 1.0)
    assert np.abs(c @ T - f).max() < 1e-11
    assert np.abs(g @ T - (1 - f)).max() < 1e-11
    assert abs(c[-1]) >= 1e-13 and c.size < 2048


def test_current_operator_generator():
    """W.square_current_hops: J = i * H_ij * (r_i - r_j) with the minimum-image displacement, Hermitian (brute force on 7 x 5)."""
    Lx, Ly = 7, 5
    n, hi, hj, hv = W.square_peierls_hops(Lx, Ly, -1.0, 0.2, 1, 7)
    H = dense_h(n, hi.numpy(), hj.numpy(), hv.numpy())
    xs, ys = np.arange(n) % Lx, np.arange(n) // Lx
    for axis, (c, L) in enumerate(((xs, Lx), (ys, Ly))):
        n2, ji, jj, jv = W.square_current_hops(Lx, Ly, axis, -1.0, 0.2, 1, 7)
        J = dense_h(n2, ji.numpy(), jj.numpy(), jv.numpy())
        d = c[:, None] - c[None, :]
        d = (d + L // 2) % L - L // 2                                # minimum image (L odd: unique)
        assert np.abs(J - 1j * H * d).max() < 1e-14
        assert np.abs(J - J.conj().T).max() < 1e-14


@pytest.mark.parametrize("beta,mu", [(1.5, 0.4), (6.0, -0.8)])
def test_corr_ac_exact_diagonalisation(oracle_mod, beta, mu):
    """corr_n = psi0^+ f(H) e^{+iHt} J_a e^{-iHt} (1 - f(H)) J_b psi0 by full diagonalisation (numpy.linalg.eigh) on a 10 x 8 square
    lattice with flux: a swapped pair of operators, a missing 1 - f, the sign of the time phase or an off-by-one in n each fail."""
    Lx, Ly, s = 10, 8, 4.8
    w = W.make_workload(4, Lx=Lx, Ly=Ly, phi_den=5)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=2).numpy()
    ja = tuple(t.numpy() for t in W.square_current_hops(Lx, Ly, 0, phi_den=5)[1:])
    jb = tuple(t.numpy() for t in W.square_current_hops(Lx, Ly, 1, phi_den=5)[1:])
    n_step = 12
    corr = oracle_mod.corr_ac(w.n_orb, on, hi, hj, hv, ja, jb, psi0, n_step, w.dt, s, beta, mu)
    H = dense_h(w.n_orb, hi, hj, hv, on)
    Ja, Jb = dense_h(w.n_orb, *ja), dense_h(w.n_orb, *jb)
    E, V = np.linalg.eigh(H)
    f = 1.0 / (np.exp(beta * (E - mu)) + 1.0)
    for b in range(2):
        p1 = V @ ((1 - f) * (V.conj().T @ (Jb @ psi0[b])))
        p2 = V @ (f * (V.conj().T @ psi0[b]))
        for n in range(n_step + 1):
            U = (V * np.exp(-1j * E * n * w.dt)) @ V.conj().T
            ref = np.vdot(U @ p2, Ja @ (U @ p1))
            assert abs(corr[b, n] - ref) < 1e-11, (b, n)
    # a full band (mu far above the spectrum): 1 - f = 0, nothing to excite
    z = oracle_mod.corr_ac(w.n_orb, on, hi, hj, hv, ja, jb, psi0[:1], 2, w.dt, s, 40.0, 3 * s)
    assert np.abs(z).max() < 1e-10


def test_corr_dp_exact_diagonalisation(oracle_mod):
    """corr_n = psi0^+ f(H) e^{+iHt} rho(q) e^{-iHt} (1 - f(H)) rho(-q) psi0 by full diagonalisation on the cubic lattice with
    disorder (N = 216); q = 0 makes rho the identity: corr_n = psi0^+ f (1 - f) psi0, constant in time."""
    w = W.make_workload(5, L=6)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=2).numpy()
    idx = np.arange(w.n_orb)
    r = np.stack([idx % 6, (idx // 6) % 6, idx // 36], axis=1).astype(np.float64)
    q = 2 * np.pi / 6 * np.array([1.0, 0.0, 2.0])
    rho = np.exp(1j * (r @ q))
    beta, mu, n_step = 0.4, 1.0, 9
    corr = oracle_mod.corr_dp(w.n_orb, on, hi, hj, hv, rho, rho.conj(), psi0, n_step, w.dt, w.rescale, beta, mu)
    H = dense_h(w.n_orb, hi, hj, hv, on)
    E, V = np.linalg.eigh(H)
    f = 1.0 / (np.exp(beta * (E - mu)) + 1.0)
    for b in range(2):
        p1 = V @ ((1 - f) * (V.conj().T @ (rho.conj() * psi0[b])))
        p2 = V @ (f * (V.conj().T @ psi0[b]))
        for n in range(n_step + 1):
            U = (V * np.exp(-1j * E * n * w.dt)) @ V.conj().T
            assert abs(corr[b, n] - np.vdot(U @ p2, rho * (U @ p1))) < 1e-11
    one = np.ones(w.n_orb, dtype=np.complex128)
    c0 = oracle_mod.corr_dp(w.n_orb, on, hi, hj, hv, one, one, psi0[:1], 4, w.dt, w.rescale, beta, mu)
    cj = V.conj().T @ psi0[0]
    assert np.abs(c0[0] - np.sum(np.abs(cj) ** 2 * f * (1 - f))).max() < 1e-11
