"""Pins of the CPU oracle against what the paper and the mathematics fix (all CPU, `-m "not gpu"`).

Each pin is independent of the oracle's own code: printed constants, closed forms, library routines
(numpy.linalg.eigh, scipy.special.jv), brute force on tiny inputs.  Numbering = SURVEY.md section 8(c).
"""
import math
import os

import numpy as np
import pytest
import scipy.special as sp

from paper_2509_26309_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def np_hops(w):
    return w.hop_i.numpy(), w.hop_j.numpy(), w.hop_val.numpy(), (None if w.onsite is None else w.onsite.numpy())


def dense_h(n, hi, hj, hv, onsite=None, hops_full=False):
    """Brute-force dense H from the hop list: H[i][j] = v, H[j][i] = conj(v)."""
    H = np.zeros((n, n), dtype=np.complex128)
    for i, j, v in zip(hi, hj, hv):
        H[i, j] += v
        if not hops_full:
            H[j, i] += np.conj(v)
    if onsite is not None:
        H[np.arange(n), np.arange(n)] += onsite
    return H


def exact_corr(H, psi0, n_step, tau, s):
    """<psi0|exp(-i H n dt)|psi0> by full diagonalisation (pin #9)."""
    E, V = np.linalg.eigh(H)
    assert np.abs(H @ V - V * E).max() < 1e-11
    wgt = np.abs(V.conj().T @ psi0) ** 2
    n = np.arange(1, n_step + 1)
    return (np.exp(-1j * np.outer(n, E) * (tau / s)) * wgt).sum(axis=1)


# ---- pin 2: Bessel -----------------------------------------------------------------------------------------
def test_bessel_printed_values(oracle_mod):
    J = oracle_mod.bessel_j(math.pi, 30)
    for line in open(os.path.join(GOLDEN, "bessel_pi.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        assert J[int(k)] == pytest.approx(float(v), rel=2e-14, abs=1e-30)


@pytest.mark.parametrize("x", [0.3, 1.0, math.pi / 2, math.pi, 2 * math.pi, 17.5, 100.0])
def test_bessel_library_and_sum_rules(oracle_mod, x):
    kmax = int(x) + 80
    J = oracle_mod.bessel_j(x, kmax)
    ref = sp.jv(np.arange(kmax + 1), x)
    assert np.abs(J - ref).max() < 5e-15
    assert J[0] + 2 * J[2::2].sum() == pytest.approx(1.0, abs=1e-14)
    assert J[0] ** 2 + 2 * (J[1:] ** 2).sum() == pytest.approx(1.0, abs=1e-14)   # unitarity of the full expansion


# ---- pins 1, 3: coefficients -------------------------------------------------------------------------------
def test_truncation_K(oracle_mod):
    assert len(oracle_mod.cheb_coeff(math.pi)) == 21
    assert len(oracle_mod.cheb_coeff(math.pi / 2)) == 16
    assert len(oracle_mod.cheb_coeff(2 * math.pi)) == 28
    assert len(oracle_mod.cheb_coeff(0.0)) == 1


@pytest.mark.parametrize("tau", [0.0, 0.7, math.pi / 2, math.pi, 2 * math.pi, 25.0])
def test_jacobi_anger_closed_form(oracle_mod, tau):
    c = oracle_mod.cheb_coeff(tau)
    x = np.linspace(-1.0, 1.0, 101)
    Tk = np.cos(np.outer(np.arange(len(c)), np.arccos(x)))
    assert np.abs(c @ Tk - np.exp(-1j * tau * x)).max() < 1e-14 * max(1.0, tau)


def test_coeff_phase_convention(oracle_mod):
    c = oracle_mod.cheb_coeff(math.pi)
    J = sp.jv(np.arange(len(c)), math.pi)
    assert c[0] == pytest.approx(J[0])
    assert c[1] == pytest.approx(-2j * J[1])
    assert c[2] == pytest.approx(-2 * J[2])
    assert c[3] == pytest.approx(2j * J[3])


# ---- pins 13-17: builder ---------------------------------------------------------------------------------
def test_csr_builder_bruteforce(oracle_mod):
    rng = np.random.default_rng(5)
    n = 23
    pairs = [(i, j) for i in range(n) for j in range(i + 1, n)]
    sel = rng.choice(len(pairs), 60, replace=False)
    hi = np.array([pairs[k][0] for k in sel], dtype=np.int32)
    hj = np.array([pairs[k][1] for k in sel], dtype=np.int32)
    flip = rng.random(60) < 0.5                      # orientation of each stored pair is arbitrary
    hi, hj = np.where(flip, hj, hi).astype(np.int32), np.where(flip, hi, hj).astype(np.int32)
    hv = rng.normal(size=60) + 1j * rng.normal(size=60)
    hv[:5] = hv[:5].real                             # real hops -> conj gives im = -0.0
    onsite = rng.normal(size=n)
    for on in (None, onsite):
        rowptr, col, val = oracle_mod.build_csr(n, on, hi, hj, hv)
        H = dense_h(n, hi, hj, hv, on)
        D = np.zeros_like(H)
        for r in range(n):
            c = col[rowptr[r]:rowptr[r + 1]]
            assert np.all(np.diff(c) > 0)            # strictly ascending columns
            D[r, c] = val[rowptr[r]:rowptr[r + 1]]
        assert np.array_equal(D, H)
        assert rowptr[-1] == 2 * 60 + (n if on is not None else 0)
        if on is not None:                           # a diagonal entry in every row
            assert all(r in col[rowptr[r]:rowptr[r + 1]] for r in range(n))
        # Hermiticity, entry by entry
        assert np.array_equal(D, D.conj().T)
    # sign bit of conj(real) is kept (compared as bits by the GPU parity test)
    rowptr, col, val = oracle_mod.build_csr(n, None, hi[:1], hj[:1], hv[:1])
    ims = val.imag
    assert sorted(np.signbit(ims).tolist()) == [False, True]


def test_csr_builder_full_list_and_errors(oracle_mod):
    hi = np.array([0, 1, 1, 2], dtype=np.int32)
    hj = np.array([1, 0, 2, 1], dtype=np.int32)
    hv = np.array([1 + 2j, 1 - 2j, 3j, -3j])
    rowptr, col, val = oracle_mod.build_csr(3, None, hi, hj, hv, hops_full=True)
    assert rowptr.tolist() == [0, 1, 3, 4] and col.tolist() == [1, 0, 2, 1]
    assert val.tolist() == [1 + 2j, 1 - 2j, 3j, -3j]
    with pytest.raises(ValueError):                  # diagonal hop is illegal
        oracle_mod.build_csr(3, None, [1], [1], [1.0])
    with pytest.raises(ValueError):                  # duplicate pair, either orientation (reading #15)
        oracle_mod.build_csr(3, None, [0, 1], [1, 0], [1.0, 1.0])
    with pytest.raises(ValueError):
        oracle_mod.build_csr(3, None, [0], [3], [1.0])
    rowptr, col, val = oracle_mod.build_csr(4, None, [], [], [])   # empty rows are legal
    assert rowptr.tolist() == [0, 0, 0, 0, 0]


def test_apply_h_matches_dense(oracle_mod):
    w = W.make_workload(4, Lx=8, Ly=6, phi_den=8)
    hi, hj, hv, _ = np_hops(w)
    on = np.linspace(-1, 1, w.n_orb)
    rng = np.random.default_rng(0)
    x = rng.normal(size=w.n_orb) + 1j * rng.normal(size=w.n_orb)
    y = oracle_mod.apply_h(w.n_orb, on, hi, hj, hv, x)
    assert np.abs(y - dense_h(w.n_orb, hi, hj, hv, on) @ x).max() < 1e-13


# ---- pin 9: exact diagonalisation on N <= 512, all three lattices ------------------------------------------
@pytest.mark.parametrize("cfg,over", [
    (1, dict(Na=16, Nb=16)),                          # honeycomb, N = 512
    (2, dict(Na=12, Nb=10)),                          # honeycomb + Anderson disorder
    (3, dict(Na=16, Nb=16)),                          # honeycomb + vacancies (irregular rows)
    (4, dict(Lx=16, Ly=16, phi_den=16)),              # square + Peierls, complex hops, s = ||H|| exactly
    (5, dict(L=8)),                                   # cubic + strong disorder, N = 512
])
def test_exact_diagonalisation(oracle_mod, cfg, over):
    w = W.make_workload(cfg, **over)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=2).numpy()
    H = dense_h(w.n_orb, hi, hj, hv, on)
    assert np.abs(np.linalg.eigvalsh(H)).max() <= w.rescale * (1 + 1e-12)
    n_step = 256
    corr, norm2 = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, n_step, w.dt, w.rescale)
    for b in range(2):
        ref = exact_corr(H, psi0[b], n_step, math.pi, w.rescale)
        assert np.abs(corr[b] - ref).max() < 1e-12
    assert np.abs(norm2 - 1).max() < 1e-12            # pin 11


def test_exact_ldos_small(oracle_mod):
    w = W.make_workload(5, L=6)
    hi, hj, hv, on = np_hops(w)
    sites = W.ldos_sites(w.n_orb, 5).numpy()
    assert len(set(sites.tolist())) == 5
    corr, _ = oracle_mod.ldos(w.n_orb, on, hi, hj, hv, sites, 64, w.dt, w.rescale)
    H = dense_h(w.n_orb, hi, hj, hv, on)
    for b, sidx in enumerate(sites):
        e = np.zeros(w.n_orb, dtype=np.complex128)
        e[sidx] = 1
        assert np.abs(corr[b] - exact_corr(H, e, 64, math.pi, w.rescale)).max() < 1e-12


def test_dimer_closed_form(oracle_mod):
    t, s = -2.7, 9.0
    corr, norm2 = oracle_mod.propagate(2, None, [0], [1], [t], np.array([[1.0, 0.0]]), 100, math.pi / s, s)
    n = np.arange(1, 101)
    assert np.abs(corr[0] - np.cos(n * math.pi * abs(t) / s)).max() < 1e-13
    assert np.abs(norm2 - 1).max() < 1e-13


# ---- pins 6, 7: semigroup and prefix -----------------------------------------------------------------------
def test_semigroup_and_prefix(oracle_mod):
    w = W.make_workload(2, Na=8, Nb=9)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=1).numpy()
    c1, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 8, w.dt, w.rescale)
    c2, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 16, w.dt / 2, w.rescale)      # K(pi/2) = 16
    assert np.abs(c1[0] - c2[0, 1::2]).max() < 1e-13
    c3, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 4, w.dt, w.rescale)
    assert np.array_equal(c3[0], c1[0, :4])
    # windowed run: restart from the state at step 4 with the same bra
    _, _, mid = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 4, w.dt, w.rescale, return_state=True)
    c4, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 4, w.dt, w.rescale, psi_start=mid)
    assert np.array_equal(c4[0], c1[0, 4:8])


# ---- pin 10: closed-form eigenstates -------------------------------------------------------------------------
def _eig_run(oracle_mod, w, psi, E, n_step=64):
    hi, hj, hv, on = np_hops(w)
    corr, norm2 = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi[None, :], n_step, w.dt, w.rescale)
    n = np.arange(1, n_step + 1)
    assert np.abs(corr[0] - np.exp(-1j * n * math.pi * E / w.rescale)).max() < 1e-12
    assert np.abs(norm2 - 1).max() < 1e-12


def test_eigenstates_honeycomb(oracle_mod):
    w = W.make_workload(1, Na=12, Nb=8)
    N = w.n_orb
    _eig_run(oracle_mod, w, np.full(N, 1 / math.sqrt(N), dtype=np.complex128), 3 * -2.7)
    stag = np.where(np.arange(N) % 2 == 0, 1.0, -1.0) / math.sqrt(N)
    _eig_run(oracle_mod, w, stag.astype(np.complex128), -3 * -2.7)


def test_eigenstates_square_and_cubic(oracle_mod):
    n, hi, hj, hv = W.square_peierls_hops(8, 6, -1.0, 0.2, 0, 1)
    w = W.Workload("sq", n, hi, hj, hv, None, 1, 1, 4.8)
    _eig_run(oracle_mod, w, np.full(n, 1 / math.sqrt(n), dtype=np.complex128), 4 * -1.0 + 4 * 0.2)
    x, y = np.arange(n) % 8, np.arange(n) // 8
    _eig_run(oracle_mod, w, ((-1.0) ** (x + y) / math.sqrt(n)).astype(np.complex128), 4.8)   # closed band edge E = s
    n, hi, hj, hv = W.cubic_hops(6, -1.0)
    w = W.Workload("cu", n, hi, hj, hv, None, 1, 1, 15.0)
    _eig_run(oracle_mod, w, np.full(n, 1 / math.sqrt(n), dtype=np.complex128), -6.0)
    k = 2 * math.pi * np.array([1, 2, 5]) / 6        # plane wave
    idx = np.arange(n)
    r = np.stack([idx % 6, (idx // 6) % 6, idx // 36], 1)
    _eig_run(oracle_mod, w, np.exp(1j * r @ k) / math.sqrt(n), 2 * -1.0 * np.cos(k).sum())


# ---- pin 25: LDOS closed form on the clean cubic lattice ----------------------------------------------------
def test_ldos_clean_cubic_closed_form(oracle_mod):
    L, s, nst = 12, 15.0, 48
    n, hi, hj, hv = W.cubic_hops(L, -1.0)
    corr, _ = oracle_mod.ldos(n, None, hi.numpy(), hj.numpy(), hv.numpy(), [0, 777], nst, math.pi / s, s, form="csr")
    q = np.arange(L)
    nn = np.arange(1, nst + 1)
    g = np.exp(-1j * np.outer(nn, 2 * -1.0 * np.cos(2 * math.pi * q / L)) * math.pi / s).mean(axis=1)
    assert np.abs(corr[0] - g ** 3).max() < 1e-13
    assert np.abs(corr[1] - g ** 3).max() < 1e-13


# ---- OpenMP row form == authoritative serial hop form ----------------------------------------------------------
@pytest.mark.parametrize("cfg,over", [(2, dict(Na=20, Nb=24)), (3, dict(Na=24, Nb=24)), (4, dict(Lx=32, Ly=24, phi_den=8)), (5, dict(L=9))])
def test_row_form_matches_hop_form(oracle_mod, cfg, over):
    w = W.make_workload(cfg, **over)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=2).numpy()
    a = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 32, w.dt, w.rescale, return_state=True)
    b = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 32, w.dt, w.rescale, form="csr", return_state=True)
    assert np.abs(a[0] - b[0]).max() < 1e-13
    assert np.abs(a[1] - b[1]).max() < 1e-13
    assert np.abs(a[2] - b[2]).max() < 1e-13


@pytest.mark.parametrize("cfg,over,tau", [(1, dict(Na=16, Nb=16), math.pi), (4, dict(Lx=16, Ly=16, phi_den=16), 2 * math.pi), (5, dict(L=8), 0.7)])
def test_row_form_exact_diagonalisation_and_window(oracle_mod, cfg, over, tau):
    """The row form (the one the full-size parity checks and the cpu_baseline use) pinned DIRECTLY, not only through the hop form:
    exact diagonalisation over 128 steps at three values of tau (other K, other flush patterns), and the windowed restart
    (psi_start) reproduces the tail of a longer run."""
    w = W.make_workload(cfg, **over)
    hi, hj, hv, on = np_hops(w)
    psi0 = w.psi0(n_state=2).numpy()
    H = dense_h(w.n_orb, hi, hj, hv, on)
    dt = tau / w.rescale
    corr, norm2, fin = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 128, dt, w.rescale, form="csr", return_state=True)
    for b in range(2):
        assert np.abs(corr[b] - exact_corr(H, psi0[b], 128, tau, w.rescale)).max() < 1e-12
    assert np.abs(norm2 - 1).max() < 1e-12
    head, _, mid = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 100, dt, w.rescale, form="csr", return_state=True)
    tail, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0, 28, dt, w.rescale, form="csr", psi_start=mid)
    assert np.abs(np.concatenate([head, tail], axis=1) - corr).max() < 1e-13


# ---- pin 27: closed-form DOS (band edges +-3|t|, van Hove peaks at +-|t|, chain 1/(pi sqrt(4t^2-E^2))) ---------
def test_dos_honeycomb_features(oracle_mod):
    w = W.make_workload(1, Na=96, Nb=96, n_step=512)
    hi, hj, hv, on = np_hops(w)
    corr, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, w.psi0(n_state=2).numpy(), 512, w.dt, w.rescale, form="csr")
    E, D = oracle_mod.dos_from_corr(corr.mean(axis=0), w.rescale)
    dE = E[1] - E[0]
    assert D.sum() * dE == pytest.approx(1.0, abs=2e-3)          # normalisation
    assert np.abs(D[np.abs(E) > 8.1 + 6 * dE]).max() < 2e-3      # band edges +-3|t| = +-8.1 eV
    assert D[np.abs(np.abs(E) - 7.9).argmin()] > 0.02            # ... and weight just inside them
    for sign in (-1, 1):                                         # van Hove peaks at +-|t| = +-2.7 eV
        m = (sign * E > 1.0) & (sign * E < 5.0)
        assert abs(E[m][D[m].argmax()] - sign * 2.7) <= 3 * dE
    # Dirac point: DOS vanishes linearly at E = 0 (single random states are noisy there, so compare averages)
    assert D[np.abs(E) < 0.15].mean() < 0.3 * D[np.abs(np.abs(E) - 1.0) < 0.15].mean()
    # closed-form per-site DOS rho(E) = (1/pi^2)(|E|/t^2) Z0^(-1/2) K(Z1/Z0) (reading #27), integrated over 1 eV bins
    def rho(e):
        x = np.abs(e) / 2.7
        za = (1 + x) ** 2 - (x ** 2 - 1) ** 2 / 4
        zb = 4 * x
        z0, z1 = np.where(x <= 1, za, zb), np.where(x <= 1, zb, za)
        return np.where(x < 3, np.abs(e) / 2.7 ** 2 / np.sqrt(z0) * sp.ellipk(np.clip(z1 / z0, 0, 1 - 1e-15)) / math.pi ** 2, 0.0)
    for lo in (-8.0, -6.0, -4.5, -2.0, -1.5, 0.5, 1.5, 3.5, 5.0, 7.0):
        fine = np.linspace(lo, lo + 1.0, 20001)[1:-1]
        ref = rho(fine).mean() * 1.0
        got = D[(E >= lo) & (E < lo + 1.0)].sum() * dE
        assert got == pytest.approx(ref, rel=0.06, abs=2e-3), (lo, got, ref)
    assert rho(np.array([1e-3]))[0] == pytest.approx(1e-3 / (math.sqrt(3) * math.pi * 2.7 ** 2), rel=1e-3)  # Dirac slope
    # second moment of the DOS = 3 t^2 (three neighbours)
    assert (D * E ** 2).sum() * dE == pytest.approx(3 * 2.7 ** 2, rel=1e-2)


def test_dos_chain_closed_form(oracle_mod):
    n, hi, hj, hv = W.chain_hops(1 << 14, -1.0)
    s = 2.5
    psi0 = W.random_phase_states(n, 4).numpy()
    corr, _ = oracle_mod.propagate(n, None, hi.numpy(), hj.numpy(), hv.numpy(), psi0, 256, math.pi / s, s, form="csr")
    E, D = oracle_mod.dos_from_corr(corr.mean(axis=0), s)
    dE = E[1] - E[0]
    for lo in np.arange(-1.5, 1.5, 0.5):              # integral of 1/(pi sqrt(4t^2-E^2)) = asin(E/2|t|)/pi
        ref = (math.asin((lo + 0.5) / 2) - math.asin(lo / 2)) / math.pi
        got = D[(E >= lo) & (E < lo + 0.5)].sum() * dE
        assert got == pytest.approx(ref, rel=0.03), (lo, got, ref)
    assert np.abs(D[np.abs(E) > 2.15]).max() < 0.02
    assert D.sum() * (E[1] - E[0]) == pytest.approx(1.0, abs=2e-3)
