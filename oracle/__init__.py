"""ORACLE (test infrastructure, not the product): ctypes front-end of oracle/tbpm_oracle.c plus numpy post-processing.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this package.
It imports nothing from paper_2509_26309_b200 (the CUDA path) and shares no code with it.  All arrays are numpy,
complex128 viewed as (re, im) float64 pairs.  See the header of tbpm_oracle.c for the algorithm and its citations.

The NEXT rows of SURVEY.md 8(f) are plain numpy on top of the C routines (quasi_eigenstates, haydock, haydock_ldos,
fermi_cheb_coeff, apply_cheb_series, corr_ac, corr_dp), each pinned in tests/test_oracle_next_pins.py by exact diagonalisation,
closed forms or brute force.  Parity unpinned: none.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "tbpm_oracle.c")
_LIB = os.path.join(_DIR, "libtbpm_oracle.so")
TOL = 1e-15   # truncation |J_k(tau)| < 1e-15 (BASELINE.json:configs[0])


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a, t=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _c128(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.complex128))


def bessel_j(x: float, kmax: int) -> np.ndarray:
    out = np.empty(kmax + 1, dtype=np.float64)
    rc = lib().oracle_bessel_j(C.c_double(x), C.c_int(kmax), _p(out))
    if rc:
        raise ValueError(f"oracle_bessel_j rc={rc}")
    return out


def cheb_coeff(tau: float, tol: float = TOL, kcap: int = 4096) -> np.ndarray:
    """complex128 [K] coefficients c_k = (2-delta_k0)(-i)^k J_k(tau)."""
    buf = np.empty(2 * kcap, dtype=np.float64)
    K = C.c_int(0)
    rc = lib().oracle_cheb_coeff(C.c_double(tau), C.c_double(tol), C.c_int(kcap), C.byref(K), _p(buf))
    if rc:
        raise ValueError(f"oracle_cheb_coeff rc={rc}")
    return buf[: 2 * K.value].view(np.complex128).copy()


def _hops(hop_i, hop_j, hop_val):
    hi = np.ascontiguousarray(np.asarray(hop_i, dtype=np.int32))
    hj = np.ascontiguousarray(np.asarray(hop_j, dtype=np.int32))
    hv = _c128(hop_val)
    assert hi.shape == hj.shape == hv.shape and hi.ndim == 1
    return hi, hj, hv


def build_csr(n_orb, onsite, hop_i, hop_j, hop_val, hops_full=False):
    """Canonical CSR (rowptr int64[n+1], col int32[nnz], val complex128[nnz])."""
    hi, hj, hv = _hops(hop_i, hop_j, hop_val)
    on = None if onsite is None else np.ascontiguousarray(np.asarray(onsite, dtype=np.float64))
    nnz = hi.size * (1 if hops_full else 2) + (n_orb if on is not None else 0)
    rowptr = np.empty(n_orb + 1, dtype=np.int64)
    col = np.empty(max(nnz, 1), dtype=np.int32)
    val = np.empty(max(nnz, 1), dtype=np.complex128)
    rc = lib().oracle_build_csr(C.c_int64(n_orb), _p(on), C.c_int64(hi.size), _p(hi, C.c_int32), _p(hj, C.c_int32),
                                _p(hv.view(np.float64)), C.c_int(int(hops_full)), _p(rowptr, C.c_int64),
                                _p(col, C.c_int32), _p(val.view(np.float64)))
    if rc:
        raise ValueError(f"oracle_build_csr rc={rc}")
    return rowptr, col[:nnz], val[:nnz]


def apply_h(n_orb, onsite, hop_i, hop_j, hop_val, x, hops_full=False):
    hi, hj, hv = _hops(hop_i, hop_j, hop_val)
    on = None if onsite is None else np.ascontiguousarray(np.asarray(onsite, dtype=np.float64))
    x = _c128(x)
    y = np.empty(n_orb, dtype=np.complex128)
    rc = lib().oracle_apply_h(C.c_int64(n_orb), _p(on), C.c_int64(hi.size), _p(hi, C.c_int32), _p(hj, C.c_int32),
                              _p(hv.view(np.float64)), C.c_int(int(hops_full)), _p(x.view(np.float64)), _p(y.view(np.float64)))
    if rc:
        raise ValueError(f"oracle_apply_h rc={rc}")
    return y


def propagate(n_orb, onsite, hop_i, hop_j, hop_val, psi0, n_step, dt, rescale, *, psi_start=None, hops_full=False,
              tol=TOL, form="hops", return_state=False):
    """corr[n_state][n_step], norm2[n_state][n_step] (and final states) for psi0[n_state][n_orb].

    form="hops": serial hop-list scatter form (authoritative).  form="csr": OpenMP row form on the canonical CSR.
    psi_start (same shape) starts the window from a later state while the bra stays psi0 (windowed parity)."""
    hi, hj, hv = _hops(hop_i, hop_j, hop_val)
    on = None if onsite is None else np.ascontiguousarray(np.asarray(onsite, dtype=np.float64))
    psi0 = np.atleast_2d(_c128(psi0))
    start = psi0 if psi_start is None else np.atleast_2d(_c128(psi_start))
    B = psi0.shape[0]
    assert psi0.shape == (B, n_orb) and start.shape == (B, n_orb)
    corr = np.zeros((B, n_step), dtype=np.complex128)
    norm2 = np.zeros((B, n_step), dtype=np.float64)
    final = np.empty((B, n_orb), dtype=np.complex128)
    if form == "csr":
        rowptr, col, val = build_csr(n_orb, on, hi, hj, hv, hops_full)
    for b in range(B):
        s, z, f = np.ascontiguousarray(start[b]), np.ascontiguousarray(psi0[b]), final[b]
        if form == "hops":
            rc = lib().oracle_propagate(C.c_int64(n_orb), _p(on), C.c_int64(hi.size), _p(hi, C.c_int32), _p(hj, C.c_int32),
                                        _p(hv.view(np.float64)), C.c_int(int(hops_full)), _p(s.view(np.float64)),
                                        _p(z.view(np.float64)), C.c_int(n_step), C.c_double(dt), C.c_double(rescale),
                                        C.c_double(tol), _p(corr[b].view(np.float64)), _p(norm2[b]), _p(f.view(np.float64)))
        elif form == "csr":
            rc = lib().oracle_propagate_csr(C.c_int64(n_orb), _p(rowptr, C.c_int64), _p(col, C.c_int32),
                                            _p(val.view(np.float64)), _p(s.view(np.float64)), _p(z.view(np.float64)),
                                            C.c_int(n_step), C.c_double(dt), C.c_double(rescale), C.c_double(tol),
                                            _p(corr[b].view(np.float64)), _p(norm2[b]), _p(f.view(np.float64)))
        else:
            raise ValueError(form)
        if rc:
            raise ValueError(f"oracle_propagate rc={rc}")
    return (corr, norm2, final) if return_state else (corr, norm2)


def ldos(n_orb, onsite, hop_i, hop_j, hop_val, sites, n_step, dt, rescale, **kw):
    """TBPM-style LDOS correlation: psi0 = e_site (reading #25), corr_n = psi_site(n dt)."""
    sites = np.asarray(sites, dtype=np.int64)
    psi0 = np.zeros((sites.size, n_orb), dtype=np.complex128)
    psi0[np.arange(sites.size), sites] = 1.0
    return propagate(n_orb, onsite, hop_i, hop_j, hop_val, psi0, n_step, dt, rescale, **kw)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def dos_from_corr(corr: np.ndarray, rescale: float):
    """DOS post-processing (NEXT-1; `Analyzer.calc_dos(corr)`, PAPER.md:980-982 gives no formula; reading #27):
    C_0 = 1, C_{-n} = conj(C_n), Hann window w_n = (1 + cos(pi n/N_t))/2 and, for tau = pi (sampling interval
    pi/s <-> energy window [-s, s]),  D(E) = (1/2s) [1 + 2 Re sum_{n=1}^{N_t} w_n C_n exp(i n pi E/s)]  on
    E_j = -s + j s/N_t, j = 0..2N_t.  Plain direct DFT, no FFT.  corr is 1-D (average over states beforehand)."""
    corr = np.asarray(corr, dtype=np.complex128).ravel()
    nt = corr.size
    n = np.arange(1, nt + 1)
    w = 0.5 * (1.0 + np.cos(np.pi * n / nt))
    E = -rescale + np.arange(2 * nt + 1) * (rescale / nt)
    ph = np.exp(1j * np.pi * np.outer(E / rescale, n))
    D = (1.0 + 2.0 * np.real(ph @ (w * corr))) / (2.0 * rescale)
    return E, D


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-3: quasi-eigenstates (QE) and the time-dependent wave function (WFT)
# ---------------------------------------------------------------------------------------------------------------------
def quasi_eigenstates(n_orb, onsite, hop_i, hop_j, hop_val, psi0, energies, n_step, dt, rescale, *, hops_full=False, form="hops"):
    """Quasi-eigenstates of the TBPM solver ("quasi-eigenstates (QE)", Table 7).

    The paper prints no formula (it defers the TBPM mathematics to the v1.3 article); reading #28:
    the Fourier transform of the time-dependent wave function at the requested energies, one-sided, Hann-windowed like
    the DOS (reading #27), NOT normalised:

        qe[b][e] = sum_{n=0}^{n_step} w_n exp(+i E_e n dt) psi_b(n dt),   w_n = (1 + cos(pi n / n_step)) / 2,  psi_b(0) = psi0[b]

    psi_b(n dt) is the oracle's own propagation, one time step at a time (oracle_propagate with n_step = 1 started from the
    previous psi), so that this function adds nothing but the plain loop above.  Returns complex128 [B][n_E][n_orb]."""
    psi0 = np.atleast_2d(_c128(psi0))
    E = np.asarray(energies, dtype=np.float64).ravel()
    B = psi0.shape[0]
    qe = np.zeros((B, E.size, n_orb), dtype=np.complex128)
    for b in range(B):
        psi = psi0[b].copy()
        for e in range(E.size):
            qe[b, e] += psi                                           # n = 0: w_0 = 1, phase 1
        for n in range(1, n_step + 1):
            _, _, fin = propagate(n_orb, onsite, hop_i, hop_j, hop_val, psi0[b], 1, dt, rescale, psi_start=psi,
                                  hops_full=hops_full, form=form, return_state=True)
            psi = fin[0]
            w = 0.5 * (1.0 + np.cos(np.pi * n / n_step))
            for e in range(E.size):
                qe[b, e] += (w * np.exp(1j * E[e] * n * dt)) * psi
    return qe


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-2: Haydock recursion (Lanczos three-term recurrence from a site) and the continued-fraction LDOS
# ---------------------------------------------------------------------------------------------------------------------
def haydock(n_orb, onsite, hop_i, hop_j, hop_val, sites, n_iter, *, hops_full=False):
    """Recursion coefficients of the Haydock method ("LDOS using Haydock recursive method"; capability list
    PAPER.md:24, 544).  The paper prints no formula; reading #29 -- the textbook recursion from |phi_0> = |site>:

        a_n = <phi_n| H |phi_n>                                   (real: H is Hermitian)
        w   = H phi_n - a_n phi_n - b_n phi_{n-1}                 (b_0 phi_{-1} = 0)
        b_{n+1} = ||w||,   phi_{n+1} = w / b_{n+1}

    Returns a [n_site][n_iter] (a_0 .. a_{n_iter-1}) and b [n_site][n_iter] (b_1 .. b_{n_iter}).  A breakdown (b = 0: the
    Krylov space is exhausted) ends the recursion of that site; the remaining entries are 0."""
    sites = np.asarray(sites, dtype=np.int64).ravel()
    a = np.zeros((sites.size, n_iter), dtype=np.float64)
    b = np.zeros((sites.size, n_iter), dtype=np.float64)
    for s, site in enumerate(sites):
        prev = np.zeros(n_orb, dtype=np.complex128)
        phi = np.zeros(n_orb, dtype=np.complex128)
        phi[site] = 1.0
        b_n = 0.0
        for n in range(n_iter):
            w = apply_h(n_orb, onsite, hop_i, hop_j, hop_val, phi, hops_full)
            a_n = float(np.vdot(phi, w).real)
            w = w - a_n * phi - b_n * prev
            b_next = float(np.sqrt(np.vdot(w, w).real))
            a[s, n], b[s, n] = a_n, b_next
            if b_next == 0.0:
                break
            prev, phi, b_n = phi, w / b_next, b_next
    return a, b


def haydock_ldos(a, b, energies, eta):
    """LDOS from the recursion coefficients: G(z) = 1 / (z - a_0 - b_1^2 / (z - a_1 - b_2^2 / (...))) at z = E + i eta,
    the fraction cut after a_{n_iter-1} (b_{n_iter} is not used: the chain is simply finite), ldos = -Im G / pi.
    a, b: [n_iter] of one site (haydock() above).  Evaluated from the bottom up."""
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    z = np.asarray(energies, dtype=np.float64).ravel() + 1j * eta
    g = np.zeros_like(z)
    for n in range(a.size - 1, -1, -1):
        tail = (b[n] ** 2) * g if n < a.size - 1 else 0.0
        g = 1.0 / (z - a[n] - tail)
    return -g.imag / np.pi


# ---------------------------------------------------------------------------------------------------------------------
# NEXT-4: AC-conductivity correlation function (Fermi-operator Chebyshev filter + current-operator matrix-vector products)
# ---------------------------------------------------------------------------------------------------------------------
def fermi_cheb_coeff(beta: float, mu: float, rescale: float, tol: float = 1e-13, n_quad: int = 8192, one_minus: bool = False) -> np.ndarray:
    """Chebyshev coefficients of the Fermi operator on [-s, s]: f(E) = 1 / (exp(beta (E - mu)) + 1) = sum_k c_k T_k(E / s),
    c_k = (2 - delta_k0) / M * sum_m f(s cos theta_m) cos(k theta_m), theta_m = pi (m + 1/2) / M (Gauss-Chebyshev quadrature, M =
    n_quad), kept up to the LAST k with |c_k| >= tol.  one_minus: the coefficients of 1 - f.  [paper silent; reading #30]"""
    m = np.arange(n_quad)
    th = np.pi * (m + 0.5) / n_quad
    x = beta * (rescale * np.cos(th) - mu)
    f = np.where(x > 0, np.exp(-np.abs(x)) / (1.0 + np.exp(-np.abs(x))), 1.0 / (1.0 + np.exp(-np.abs(x))))
    kmax = n_quad // 4
    c = np.array([(1.0 if k == 0 else 2.0) / n_quad * np.sum(f * np.cos(k * th)) for k in range(kmax)])
    big = np.nonzero(np.abs(c) >= tol)[0]
    K = int(big[-1]) + 1 if big.size else 1
    c = c[:K].copy()
    if one_minus:
        c = -c
        c[0] += 1.0
    return c


def apply_cheb_series(n_orb, onsite, hop_i, hop_j, hop_val, coeff, rescale, x, hops_full=False):
    """y = sum_k coeff[k] T_k(H / s) x by the forward recurrence T_0 = x, T_1 = H' x, T_{k+1} = 2 H' T_k - T_{k-1} (the loop of
    PAPER.md:437-443 with other coefficients), H applied by the oracle's hop-list routine."""
    coeff = np.asarray(coeff)
    t0 = _c128(x).copy()
    y = coeff[0] * t0
    if coeff.size > 1:
        t1 = apply_h(n_orb, onsite, hop_i, hop_j, hop_val, t0, hops_full) / rescale
        y = y + coeff[1] * t1
        for k in range(2, coeff.size):
            t2 = (2.0 / rescale) * apply_h(n_orb, onsite, hop_i, hop_j, hop_val, t1, hops_full) - t0
            y = y + coeff[k] * t2
            t0, t1 = t1, t2
    return y


def corr_ac(n_orb, onsite, hop_i, hop_j, hop_val, ja_hops, jb_hops, psi0, n_step, dt, rescale, beta, mu):
    """AC-conductivity correlation of TBPM ("AC conductivity (AC)" is a solver function of the paper, Table 7
    PAPER.md:1744; the current operator acts through a sparse matrix-vector product; no formula is printed).
    DESIGN.md reading #30, with f the Fermi operator and J_a, J_b the current-operator matrices (given as hop lists, Hermitian):

        psi1(0) = [1 - f(H)] J_b psi0,   psi2(0) = f(H) psi0,   psi_i(t) = exp(-i H t) psi_i(0)
        corr[b][n] = < psi2(n dt) | J_a | psi1(n dt) >,   n = 0 .. n_step

    f(H) and 1 - f(H) by their Chebyshev series (fermi_cheb_coeff), the time evolution by the oracle's own propagation one step at a
    time.  ja_hops / jb_hops = (hop_i, hop_j, hop_val) of the two current operators (each conjugate pair once).  Returns complex128
    [B][n_step + 1]."""
    psi0 = np.atleast_2d(_c128(psi0))
    cf = fermi_cheb_coeff(beta, mu, rescale)
    cg = fermi_cheb_coeff(beta, mu, rescale, one_minus=True)
    out = np.zeros((psi0.shape[0], n_step + 1), dtype=np.complex128)
    for b in range(psi0.shape[0]):
        phi = apply_h(n_orb, None, *jb_hops, psi0[b])
        p1 = apply_cheb_series(n_orb, onsite, hop_i, hop_j, hop_val, cg, rescale, phi)
        p2 = apply_cheb_series(n_orb, onsite, hop_i, hop_j, hop_val, cf, rescale, psi0[b])
        for n in range(n_step + 1):
            if n > 0:
                _, _, fin = propagate(n_orb, onsite, hop_i, hop_j, hop_val, p1, 1, dt, rescale, psi_start=p1, return_state=True)
                p1 = fin[0]
                _, _, fin = propagate(n_orb, onsite, hop_i, hop_j, hop_val, p2, 1, dt, rescale, psi_start=p2, return_state=True)
                p2 = fin[0]
            out[b, n] = np.vdot(p2, apply_h(n_orb, None, *ja_hops, p1))
    return out


def corr_dp(n_orb, onsite, hop_i, hop_j, hop_val, rho_a, rho_b, psi0, n_step, dt, rescale, beta, mu):
    """Dynamic-polarisation correlation of TBPM ("dynamic polarizability (DP)", Table 7; no formula
    printed).  DESIGN.md reading #31: the scheme of corr_ac with the DIAGONAL density operators rho(q) = diag(exp(i q.r_i)) in place
    of the current operators -- rho_a, rho_b are complex128 [n_orb] (the caller passes rho_b = rho(-q), rho_a = rho(q)):

        psi1(0) = [1 - f(H)] (rho_b * psi0),   psi2(0) = f(H) psi0,   corr[b][n] = < psi2(n dt) | rho_a * psi1(n dt) >,  n = 0 .. n_step."""
    psi0 = np.atleast_2d(_c128(psi0))
    ra, rb = _c128(rho_a), _c128(rho_b)
    cf = fermi_cheb_coeff(beta, mu, rescale)
    cg = fermi_cheb_coeff(beta, mu, rescale, one_minus=True)
    out = np.zeros((psi0.shape[0], n_step + 1), dtype=np.complex128)
    for b in range(psi0.shape[0]):
        p1 = apply_cheb_series(n_orb, onsite, hop_i, hop_j, hop_val, cg, rescale, rb * psi0[b])
        p2 = apply_cheb_series(n_orb, onsite, hop_i, hop_j, hop_val, cf, rescale, psi0[b])
        for n in range(n_step + 1):
            if n > 0:
                _, _, fin = propagate(n_orb, onsite, hop_i, hop_j, hop_val, p1, 1, dt, rescale, psi_start=p1, return_state=True)
                p1 = fin[0]
                _, _, fin = propagate(n_orb, onsite, hop_i, hop_j, hop_val, p2, 1, dt, rescale, psi_start=p2, return_state=True)
                p2 = fin[0]
            out[b, n] = np.vdot(p2, ra * p1)
    return out
