"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs (`-m gpu`).

Bar (BASELINE.json:north_star): hopping-to-sparse index build bit-exact; max |delta corr| <= 1e-10 absolute in fp64;
|norm2 - 1| <= 1e-12.  Small cases compare every element against the authoritative serial oracle; the full-size
configs use prefix parity on a sample of states (the first m steps do not depend on n_step, reading #7) against the
OpenMP row form of the oracle (itself pinned to the serial form), closed-form eigenstates at full size, and the
norm invariant.
"""
import math
import os

import numpy as np
import pytest
import torch

from paper_2509_26309_b200 import tbpm, workloads as W

pytestmark = pytest.mark.gpu

CORR_TOL = 1e-10     # north_star
NORM_TOL = 1e-12     # north_star


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def to_np(w):
    return (w.hop_i.cpu().numpy(), w.hop_j.cpu().numpy(), w.hop_val.cpu().numpy(),
            None if w.onsite is None else w.onsite.cpu().numpy())


def assert_csr_bit_exact(H, oracle_mod, w, hops_full=False):
    hi, hj, hv, on = to_np(w)
    orow, ocol, oval = oracle_mod.build_csr(w.n_orb, on, hi, hj, hv, hops_full)
    rowptr, col, val = tbpm.tbpm_export_csr(H)
    torch.cuda.synchronize()
    assert np.array_equal(rowptr.cpu().numpy(), orow)
    assert np.array_equal(col.cpu().numpy(), ocol)
    assert np.array_equal(val.cpu().numpy().view(np.uint64), oval.view(np.uint64))   # raw 64-bit patterns (-0.0 matters)


# ---------------------------------------------------------------------------------------------------------------------
# a0: builder
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,over", [
    (1, {}),                                           # config 1 at full size
    (2, dict(Na=96, Nb=70)),                           # with on-site diagonal
    (3, dict(Na=128, Nb=96)),                          # vacancies: rows of 0..3 entries, empty rows
    (4, dict(Lx=64, Ly=48, phi_den=32)),               # complex values, 8 per row
    (5, dict(L=17)),                                   # 7 per row incl. diagonal, ragged tail (4913 rows)
])
@pytest.mark.parametrize("flags", [0, tbpm.TBPM_NO_TABLE])
def test_build_bit_exact(dev, oracle_mod, cfg, over, flags):
    w = W.make_workload(cfg, device=dev, **over)
    # the result must not depend on the order of the list
    perm = torch.randperm(w.n_hop, generator=torch.Generator().manual_seed(cfg)).to(dev)
    w.hop_i, w.hop_j, w.hop_val = w.hop_i[perm].contiguous(), w.hop_j[perm].contiguous(), w.hop_val[perm].contiguous()
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val, flags | tbpm.TBPM_VALIDATE)
    assert H.nnz == w.nnz
    assert_csr_bit_exact(H, oracle_mod, w)
    hi, hj, hv, on = to_np(w)
    rowsum = np.zeros(w.n_orb)
    np.add.at(rowsum, hi, np.abs(hv))
    np.add.at(rowsum, hj, np.abs(hv))
    if on is not None:
        rowsum += np.abs(on)
    assert H.gershgorin == pytest.approx(rowsum.max(), rel=1e-12)
    assert tbpm.tbpm_check_bound(H, w.rescale) == tbpm.TBPM_OK        # config 4: equality is allowed
    assert tbpm.tbpm_check_bound(H, 0.5 * w.rescale) == tbpm.TBPM_EBOUND
    if flags & tbpm.TBPM_NO_TABLE:
        assert H.n_table == 0
    else:
        # v and conj(v) share a table entry: distinct (re, |im|) bit patterns
        assert H.n_table == len(set(zip(np.ascontiguousarray(hv.real).view(np.uint64).tolist(),
                                        np.abs(hv.imag).view(np.uint64).tolist())))


def test_build_edge_cases(dev, oracle_mod):
    i32 = lambda a: torch.tensor(a, dtype=torch.int32, device=dev)
    c128 = lambda a: torch.tensor(a, dtype=torch.complex128, device=dev)
    # both orientations supplied by the caller
    w = W.Workload("full", 3, i32([0, 1, 1, 2]), i32([1, 0, 2, 1]), c128([1 + 2j, 1 - 2j, 3j, -3j]), None, 1, 1, 1.0)
    H = tbpm.tbpm_build(3, None, w.hop_i, w.hop_j, w.hop_val, tbpm.TBPM_HOPS_FULL)
    assert_csr_bit_exact(H, oracle_mod, w, hops_full=True)
    # no hops at all, with and without diagonal; zero orbitals
    e = W.Workload("empty", 5, i32([]), i32([]), c128([]), None, 1, 1, 1.0)
    H = tbpm.tbpm_build(5, None, e.hop_i, e.hop_j, e.hop_val)
    assert H.nnz == 0 and tbpm.tbpm_export_csr(H)[0].tolist() == [0] * 6
    e.onsite = torch.linspace(-1, 1, 5, dtype=torch.float64, device=dev)
    H = tbpm.tbpm_build(5, e.onsite, e.hop_i, e.hop_j, e.hop_val)
    assert_csr_bit_exact(H, oracle_mod, e)
    H = tbpm.tbpm_build(0, None, e.hop_i, e.hop_j, e.hop_val)
    assert H.nnz == 0 and H.n_orb == 0
    # one long row (star graph): max_row_nnz, sorting of a long segment
    n = 3000
    star = W.Workload("star", n, i32(list(range(1, n))[::-1]), i32([0] * (n - 1)),
                      torch.full((n - 1,), 0.001 + 0.002j, dtype=torch.complex128, device=dev), None, 1, 1, 10.0)
    H = tbpm.tbpm_build(n, None, star.hop_i, star.hop_j, star.hop_val)
    assert H.max_row_nnz == n - 1
    assert_csr_bit_exact(H, oracle_mod, star)
    sp0 = star.psi0(device=dev, n_state=2)                            # a row of 2,999 entries on the general kernel
    sc, sn, _ = tbpm.tbpm_propagate(H, sp0, 4, star.dt, star.rescale)
    shi, shj, shv, _ = to_np(star)
    sref, _ = oracle_mod.propagate(n, None, shi, shj, shv, sp0.cpu().numpy(), 4, star.dt, star.rescale)
    assert np.abs(sc.cpu().numpy() - sref).max() <= CORR_TOL and np.abs(sn.cpu().numpy() - 1).max() <= NORM_TOL
    # errors
    for hi, hj, code in (([1], [1], tbpm.TBPM_EDIAG), ([0, 1], [1, 0], tbpm.TBPM_EDUP), ([0, 0], [1, 1], tbpm.TBPM_EDUP),
                         ([0], [3], tbpm.TBPM_EINDEX), ([-1], [2], tbpm.TBPM_EINDEX)):
        with pytest.raises(tbpm.TbpmError) as ei:
            tbpm.tbpm_build(3, None, i32(hi), i32(hj), c128([1.0] * len(hi)), tbpm.TBPM_VALIDATE)
        assert ei.value.code == code


def test_table_overflow_falls_back_to_full_values(dev, oracle_mod):
    # > 32768 distinct hopping values (v and conj v count once): the kernels must read complex128 values from the canonical CSR
    n = 70001
    i = torch.arange(n - 1, dtype=torch.int32, device=dev)
    vals = torch.complex(torch.linspace(0.1, 0.9, n - 1, dtype=torch.float64, device=dev),
                         torch.linspace(-0.3, 0.3, n - 1, dtype=torch.float64, device=dev))
    w = W.Workload("many", n, i, i + 1, vals, None, 2, 8, 2.0)
    H = tbpm.tbpm_build(n, None, w.hop_i, w.hop_j, w.hop_val)
    assert H.n_table == 0
    assert_csr_bit_exact(H, oracle_mod, w)
    psi0 = w.psi0(device=dev)
    corr, norm2, _ = tbpm.tbpm_propagate(H, psi0, 8, w.dt, w.rescale)
    hi, hj, hv, on = to_np(w)
    ref, _ = oracle_mod.propagate(n, on, hi, hj, hv, psi0.cpu().numpy(), 8, w.dt, w.rescale)
    assert np.abs(corr.cpu().numpy() - ref).max() <= CORR_TOL


# ---------------------------------------------------------------------------------------------------------------------
# a1-a7: propagate, every element against the serial oracle
# ---------------------------------------------------------------------------------------------------------------------
def run_parity(dev, oracle_mod, w, n_state, n_step, flags=0, dt=None, check_state=True, options=None):
    dt = w.dt if dt is None else dt
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val, flags)
    for opt, value in (options or {}).items():
        tbpm.tbpm_set_option(H, opt, value)
    corr, norm2, ws = tbpm.tbpm_propagate(H, psi0, n_step, dt, w.rescale)
    hi, hj, hv, on = to_np(w)
    ref, refn, reff = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0.cpu().numpy(), n_step, dt, w.rescale, return_state=True)
    assert np.abs(corr.cpu().numpy() - ref).max() <= CORR_TOL
    assert np.abs(norm2.cpu().numpy() - refn).max() <= NORM_TOL
    assert np.abs(norm2.cpu().numpy() - 1).max() <= NORM_TOL
    if check_state:
        for b in sorted({0, n_state - 1}):
            got = tbpm.tbpm_get_state(H, ws, b).cpu().numpy()
            assert np.abs(got - reff[b]).max() <= 1e-12
    return H, psi0, corr, norm2


def test_config1_full_length(dev, oracle_mod):
    """BASELINE.json:configs[0] exactly: honeycomb 64x64, 1 state, 256 steps, s = 9, tau = pi."""
    w = W.make_workload(1, device=dev)
    H, _, corr, _ = run_parity(dev, oracle_mod, w, 1, 256)
    assert corr.shape == (1, 256)
    assert H.n_table == 1                                            # t and conj(t) = (t, -0.0) share the entry
    assert tbpm.tbpm_last_launch_count(H) == 2                       # state set-up + ONE cluster launch for all 256 steps (k_small_steps)
    tbpm.tbpm_set_option(H, tbpm.TBPM_OPT_KERNEL, 2)                 # the same on the launch-per-term path
    psi0 = w.psi0(device=dev, n_state=1)
    c2, n2, _ = tbpm.tbpm_propagate(H, psi0, 256, w.dt, w.rescale)
    assert tbpm.tbpm_last_launch_count(H) == 256 * 21 + 1            # 20 terms + 1 final reduction per step, + set-up
    assert (c2 - corr).abs().max() <= 1e-13 and np.abs(n2.cpu().numpy() - 1).max() <= NORM_TOL


@pytest.mark.parametrize("cfg,over,n_state,n_step", [
    (2, dict(Na=96, Nb=70), 4, 24),                                  # 13440 rows: several blocks + ragged tail
    (2, dict(Na=33, Nb=35), 3, 9),                                   # 3 states -> padded tile of 4
    (3, dict(Na=128, Nb=96), 1, 24),                                 # irregular rows 0..3, empty rows
    (3, dict(Na=100, Nb=60), 2, 7),
    (4, dict(Lx=64, Ly=48, phi_den=32), 8, 24),                      # complex hops, SpMM tile of 8, s = ||H||
    (4, dict(Lx=32, Ly=24, phi_den=8), 5, 6),                        # 5 states -> padded tile of 8
    (5, dict(L=17), 32, 12),                                         # 4 tiles of 8
    (5, dict(L=12), 11, 5),                                          # tile of 8 + padded tile of 4
    (5, dict(L=32), 8, 6),                                           # plane stride 1024 = 8 tiles: the builder's lattice walk
])
@pytest.mark.parametrize("flags", [0, tbpm.TBPM_NO_TABLE])
def test_small_configs_every_element(dev, oracle_mod, cfg, over, n_state, n_step, flags):
    w = W.make_workload(cfg, device=dev, **over)
    run_parity(dev, oracle_mod, w, n_state, n_step, flags)


# lattices on which the lattice kernels apply (tiles of 8 states): term_l3.cu on three-dimensional lattices whose line is a
# multiple of 32 rows and whose plane a multiple of 4 lines; term_rw.cu when the largest stride is a multiple of 128 rows
RW_CASES = [
    (5, dict(L=32), 8, 7),                                           # cubic 32^3: one tile per line, 8 tile rows per plane, diagonal
    (5, dict(L=32, W=0.0), 11, 5),                                   # no diagonal; tile of 8 + padded tile of 4 (phased kernel)
    (5, dict(L=64), 8, 3),                                           # cubic 64^3: two tiles per line, runs of 64 planes
    (5, dict(L=16, W=0.0), 16, 6),                                   # cubic 16^3 (line of 16 rows: term_rw only, W = 256), two tiles
    (4, dict(Lx=128, Ly=24, phi_den=32), 8, 9),                      # square + flux: W = 128, 8 entries, table of values
    (4, dict(Lx=256, Ly=12, phi_den=64), 13, 5),                     # W = 256: two tiles per line; tile of 8 + padded tile of 8
]


@pytest.mark.parametrize("cfg,over,n_state,n_step", RW_CASES)
@pytest.mark.parametrize("kernel", [0, 1, 2, 3, 4])
def test_lattice_kernels_agree_with_oracle(dev, oracle_mod, cfg, over, n_state, n_step, kernel):
    """The same lattices on the lattice kernels (default: term_l3 where it applies, else term_rw; on the square lattice two terms
    per sweep, term_sq2 -- one term per sweep, term_sq, with TBPM_OPT_KERNEL = 4), the general kernel
    (TBPM_OPT_KERNEL = 1), the phased kernel (2) and term_rw alone (3): every element against the serial oracle; rows on the
    seams of the periodic lattice are gathered entry by entry inside the lattice kernels."""
    w = W.make_workload(cfg, device=dev, **over)
    run_parity(dev, oracle_mod, w, n_state, n_step, options={tbpm.TBPM_OPT_KERNEL: kernel})


def test_lattice_kernels_rows_off_the_lattice(dev, oracle_mod):
    """Matrices that only RESEMBLE a lattice.  (i) Cubic 32^3 with two bonds rewired (a-b, c-d -> a-d, c-b): every row still has six
    entries, four rows are off the lattice -- term_l3 keeps running and gathers the warps that hold them entry by entry through
    ocol.  (ii) Square lattice with flux where ONE hopping value is changed: the per-line table no longer describes every row, the
    builder must not certify it (lattice kind 0) and the rolling-window kernel takes over."""
    w = W.make_workload(5, device=dev, L=32)
    hi, hj = w.hop_i.clone(), w.hop_j.clone()
    h1, h2 = 12345, 54321 + 32768                                    # an x-bond and a y-bond far apart
    hj[h1], hj[h2] = w.hop_j[h2], w.hop_j[h1]
    w.hop_i, w.hop_j = hi, hj
    H, _, _, _ = run_parity(dev, oracle_mod, w, 8, 5)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_CUBIC
    w = W.make_workload(4, device=dev, Lx=128, Ly=24, phi_den=32)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_SQUARE8
    w.hop_val = w.hop_val.clone()
    w.hop_val[777] = w.hop_val[777] * 0.5
    H, _, _, _ = run_parity(dev, oracle_mod, w, 8, 5)
    assert H.lattice_kind == 0


@pytest.mark.parametrize("tau_scale", [1.0, 0.9, 0.5, 0.3, 0.05])
def test_two_terms_per_sweep(dev, oracle_mod, tau_scale):
    """term_sq2.cu (two Chebyshev terms per launch on the square lattice of cfg4): time steps whose series have an even and an odd
    number of terms (K = 21, 20, 16, 14, 9: a leading single term when K - 1 is odd, psi' touched every second pair), a lattice of
    three tiles per line and more lines than one run holds, 16 states = two tiles; against the oracle, against the one-term-per-sweep
    path (TBPM_OPT_KERNEL = 4), and by the launch count (the pairs really ran)."""
    w = W.make_workload(4, device=dev, Lx=384, Ly=150, phi_den=128)
    dt = w.dt * tau_scale
    K = len(tbpm.tbpm_cheb_coeff(w.rescale * dt))
    n_step, n_state = 4, 16
    H, psi0, corr, norm2 = run_parity(dev, oracle_mod, w, n_state, n_step, dt=dt)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_SQUARE8
    n_launch = (K - 1) // 2 + (K - 1) % 2                               # pairs (+ a leading single term)
    assert tbpm.tbpm_last_launch_count(H) == 2 * (1 + n_step * (n_launch + 1))   # per tile: set-up + per step the launches + reduction
    tbpm.tbpm_set_option(H, tbpm.TBPM_OPT_KERNEL, 4)
    c1, n1, _ = tbpm.tbpm_propagate(H, psi0, n_step, dt, w.rescale)
    assert tbpm.tbpm_last_launch_count(H) == 2 * (1 + n_step * K)
    assert (c1 - corr).abs().max().item() <= 1e-13 and (n1 - norm2).abs().max().item() <= 1e-13
    # a caller workspace without the two extra vectors: the call falls back to one term per sweep instead of failing
    tbpm.tbpm_set_option(H, tbpm.TBPM_OPT_KERNEL, 0)
    full = tbpm.tbpm_propagate_bytes(H, n_state)
    small = torch.empty(full - 2 * 16 * w.n_orb * 8, dtype=torch.uint8, device=dev)
    c2, n2, _ = tbpm.tbpm_propagate(H, psi0, n_step, dt, w.rescale, workspace=small)
    assert tbpm.tbpm_last_launch_count(H) == 2 * (1 + n_step * K)
    assert torch.equal(c2.view(torch.float64), c1.view(torch.float64))


@pytest.mark.parametrize("Lx,Ly,phi_den", [(256, 70, 64), (128, 40, 32)])                # two tiles per line / one (both line ends in one tile)
@pytest.mark.parametrize("tau_scale", [1.0, 0.45])
def test_two_terms_per_sweep_with_diagonal(dev, oracle_mod, tau_scale, Lx, Ly, phi_den):
    """The pair kernel with a real diagonal (square lattice + flux + Anderson disorder: the diagonal of 132 rows per line rides in
    the y stage, also on the first pair, which has no T_{k-2}): even and odd numbers of terms, two tiles of states, both paths."""
    n, hi, hj, hv = W.square_peierls_hops(Lx, Ly, -1.0, 0.2, 1, phi_den, dev)
    w = W.Workload("square-flux-anderson", n, hi, hj, hv, W.anderson_onsite(n, 3.0, device=dev), 16, 5, 6.4)
    dt = w.dt * tau_scale
    K = len(tbpm.tbpm_cheb_coeff(w.rescale * dt))
    H, psi0, corr, norm2 = run_parity(dev, oracle_mod, w, 16, 5, dt=dt)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_SQUARE8
    assert tbpm.tbpm_last_launch_count(H) == 2 * (1 + 5 * ((K - 1) // 2 + (K - 1) % 2 + 1))
    tbpm.tbpm_set_option(H, tbpm.TBPM_OPT_KERNEL, 4)
    c1, n1, _ = tbpm.tbpm_propagate(H, psi0, 5, dt, w.rescale)
    assert tbpm.tbpm_last_launch_count(H) == 2 * (1 + 5 * K)
    assert (c1 - corr).abs().max().item() <= 1e-13 and (n1 - norm2).abs().max().item() <= 1e-13


def test_two_terms_per_sweep_complex_inline_hops(dev, oracle_mod):
    """The builder certifies whether the hops ALONG a line are real (Landau gauge: they are; the pair kernel then spends two FMAs on
    them instead of four).  Here they carry a constant phase -- still a function of the in-line position only, so the square-lattice
    kernels run, but on their general (complex) variant; with and without diagonal."""
    n, hi, hj, hv = W.square_peierls_hops(256, 40, -1.0, 0.2, 1, 64, dev)
    inline = (hi // 256) == (hj // 256)
    hv = torch.where(inline, hv * torch.exp(torch.tensor(0.3j, dtype=torch.complex128, device=dev)), hv)
    for onsite in (None, W.anderson_onsite(n, 2.0, device=dev)):
        w = W.Workload("square-flux-twisted", n, hi, hj, hv, onsite, 8, 5, 6.0)
        H, psi0, corr, norm2 = run_parity(dev, oracle_mod, w, 8, 5)
        assert H.lattice_kind == tbpm.TBPM_LATTICE_SQUARE8
        assert tbpm.tbpm_last_launch_count(H) == 1 + 5 * 11


def test_two_terms_per_sweep_ldos_and_determinism(dev, oracle_mod):
    """The pair path under tbpm_ldos (unit initial vectors) and twice in a row: bit-identical."""
    w = W.make_workload(4, device=dev, Lx=128, Ly=40, phi_den=32)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    sites = W.ldos_sites(w.n_orb, 8)
    c1, n1, _ = tbpm.tbpm_ldos(H, sites, 6, w.dt, w.rescale)
    assert tbpm.tbpm_last_launch_count(H) == 1 + 6 * 11                  # unit-vector set-up + 6 x (10 pairs + reduction)
    c2, n2, _ = tbpm.tbpm_ldos(H, sites, 6, w.dt, w.rescale)
    assert torch.equal(c1.view(torch.float64), c2.view(torch.float64)) and torch.equal(n1, n2)
    psi0 = torch.zeros((8, w.n_orb), dtype=torch.complex128, device=dev)
    psi0[torch.arange(8), torch.as_tensor(sites, device=dev)] = 1.0
    hi, hj, hv, on = to_np(w)
    ref, refn = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0.cpu().numpy(), 6, w.dt, w.rescale)[:2]
    assert np.abs(c1.cpu().numpy() - ref).max() <= CORR_TOL and np.abs(n1.cpu().numpy() - refn).max() <= NORM_TOL


def test_short_row_kernel(dev, oracle_mod):
    """term_n16.cu (tiles of one state, rows of <= 4 entries, one real value, 16-bit column offsets): honeycomb with vacancies (rows of
    0-3 entries, periodic wrap entries stored modulo n_orb), the clean honeycomb lattice with on-site disorder (diagonal), a ring (only
    +-1 neighbours: every gather is a warp shuffle except at the warp ends and across the ends of the ring), a square lattice with four
    real neighbours (4 slots); and a lattice too wide for 16-bit offsets, which must stay on the phased kernel."""
    w = W.make_workload(3, device=dev, Na=160, Nb=120)
    H, _, _, _ = run_parity(dev, oracle_mod, w, 1, 12)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_NEAR16
    w = W.make_workload(2, device=dev, Na=150, Nb=131)
    H, _, _, _ = run_parity(dev, oracle_mod, w, 1, 9)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_NEAR16
    n = 70001
    i = torch.arange(n, device=dev, dtype=torch.int32)
    w = W.Workload("ring", n, i, ((i + 1) % n).to(torch.int32), torch.full((n,), -1.0, dtype=torch.complex128, device=dev), None, 1, 10, 2.5)
    H, _, _, _ = run_parity(dev, oracle_mod, w, 1, 10)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_NEAR16
    n, hi, hj, hv = W.square_peierls_hops(320, 90, -1.0, 0.0, 1, 32, dev)
    keep = hv.abs() > 0
    w = W.Workload("square-nn", n, hi[keep].contiguous(), hj[keep].contiguous(), torch.full((int(keep.sum()),), -1.0, dtype=torch.complex128, device=dev),
                   W.anderson_onsite(n, 2.0, device=dev), 1, 8, 5.5)
    H, _, _, _ = run_parity(dev, oracle_mod, w, 1, 8)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_NEAR16
    n, hi, hj, hv = W.square_peierls_hops(40000, 3, -1.0, 0.0, 1, 32, dev)      # line of 40000 rows: the line neighbours do not fit 16 bits
    keep = hv.abs() > 0
    w = W.Workload("square-wide", n, hi[keep].contiguous(), hj[keep].contiguous(), torch.full((int(keep.sum()),), -1.0, dtype=torch.complex128, device=dev),
                   None, 1, 4, 4.5)
    H, _, _, _ = run_parity(dev, oracle_mod, w, 1, 4)
    assert H.lattice_kind == 0


def test_anisotropic_box_lattice(dev, oracle_mod):
    """A 64 x 8 x 12 box (line of 64 rows = two tiles, plane of 8 lines = two tile rows, 12 planes: runs shorter than 64) with
    Anderson disorder: the three-dimensional lattice kernel away from the cube, 16 states = two tiles."""
    Lx, Ly, Lz = 64, 8, 12
    z = torch.arange(Lz, device=dev).view(Lz, 1, 1); y = torch.arange(Ly, device=dev).view(1, Ly, 1); x = torch.arange(Lx, device=dev).view(1, 1, Lx)
    idx = lambda zz, yy, xx: ((zz * Ly + yy) * Lx + xx).expand(Lz, Ly, Lx).reshape(-1)
    src = idx(z, y, x)
    hop_i = torch.cat([src, src, src]).to(torch.int32)
    hop_j = torch.cat([idx(z, y, (x + 1) % Lx), idx(z, (y + 1) % Ly, x), idx((z + 1) % Lz, y, x)]).to(torch.int32)
    n = Lx * Ly * Lz
    w = W.Workload("box", n, hop_i, hop_j, torch.full((3 * n,), -1.0, dtype=torch.complex128, device=dev),
                   W.anderson_onsite(n, 4.0, device=dev), 16, 6, 8.5)
    H, _, _, _ = run_parity(dev, oracle_mod, w, 16, 6)
    assert H.lattice_kind == tbpm.TBPM_LATTICE_CUBIC


def test_square_nn_lattice_rolling_window(dev, oracle_mod):
    """4 entries per row (t' = 0): the third instantiated shape of term_rw, with one real hopping value and with phases."""
    n, hi, hj, hv = W.square_peierls_hops(128, 20, -1.0, 0.0, 1, 32, dev)
    keep = hv.abs() > 0                                              # drop the t' = 0 entries
    w = W.Workload("square-nn-flux", n, hi[keep].contiguous(), hj[keep].contiguous(), hv[keep].contiguous(), None, 8, 6, 4.0)
    run_parity(dev, oracle_mod, w, 8, 6)
    w.hop_val = torch.full_like(w.hop_val, -1.0)
    run_parity(dev, oracle_mod, w, 8, 6)


@pytest.mark.parametrize("radius,n_phase,n_state", [
    (2, 1, 8), (2, 16, 1), (2, 1, 4),                                # 12 entries per row: phased kernel, chunked rows
    (4, 8, 8), (4, 1, 2),                                            # 48 entries: phased kernel at 8 states, general kernel at 2
    (5, 4, 8), (5, 32, 3),                                           # 80 entries: general kernel with the value table
])
@pytest.mark.parametrize("diag", [False, True])
def test_long_rows(dev, oracle_mod, radius, n_phase, n_state, diag):
    """Rows of 12 / 48 / 80 entries (hops to every site within a radius; BASELINE.json's configs stop at 8): covers the
    chunked row loop of term_ph.cuh, its stage-size dispatch, and k_cheb_term<..., TABLE = true> on long rows."""
    n, hi, hj, hv, row_sum = W.square_range_hops(32, 24, radius, n_phase, dev)
    onsite = torch.linspace(-0.5, 0.5, n, dtype=torch.float64, device=dev) if diag else None
    w = W.Workload(f"range{radius}", n, hi, hj, hv, onsite, n_state, 5, row_sum + 0.5)
    H, _, _, _ = run_parity(dev, oracle_mod, w, n_state, 5)
    assert H.max_row_nnz == {2: 12, 4: 48, 5: 80}[radius] + int(diag) and H.n_table > 0
    run_parity(dev, oracle_mod, w, n_state, 3, tbpm.TBPM_NO_TABLE)


@pytest.mark.parametrize("cfg,over,n_state,n_step", [
    (2, dict(Na=96, Nb=70), 4, 8), (3, dict(Na=100, Nb=60), 2, 7), (4, dict(Lx=64, Ly=48, phi_den=32), 8, 6), (5, dict(L=17), 11, 5),
])
def test_general_kernel_every_shape(dev, oracle_mod, cfg, over, n_state, n_step):
    """TBPM_OPT_KERNEL = 1: every term on k_cheb_term (the path of tables > 32768 values, tiles of 16 / 32 states, long rows)."""
    w = W.make_workload(cfg, device=dev, **over)
    run_parity(dev, oracle_mod, w, n_state, n_step, options={tbpm.TBPM_OPT_KERNEL: 1})


@pytest.mark.parametrize("tile", [1, 2, 4, 16, 32])
def test_other_tile_widths(dev, oracle_mod, tile):
    w = W.make_workload(5, device=dev, L=13)
    run_parity(dev, oracle_mod, w, 35 if tile >= 16 else 7, 6, options={tbpm.TBPM_OPT_TILE: tile})
    w = W.make_workload(4, device=dev, Lx=48, Ly=32, phi_den=16)
    run_parity(dev, oracle_mod, w, 33 if tile == 32 else 6, 5, tbpm.TBPM_NO_TABLE, options={tbpm.TBPM_OPT_TILE: tile})


def test_options_and_get_state_checks(dev):
    w = W.make_workload(2, device=dev, Na=24, Nb=20)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    for opt, bad in ((tbpm.TBPM_OPT_TILE, 3), (tbpm.TBPM_OPT_TILE, 64), (tbpm.TBPM_OPT_KERNEL, 7), (99, 0)):
        with pytest.raises(tbpm.TbpmError) as ei:
            tbpm.tbpm_set_option(H, opt, bad)
        assert ei.value.code == tbpm.TBPM_EINVAL
    psi0 = w.psi0(device=dev, n_state=3)
    _, _, ws = tbpm.tbpm_propagate(H, psi0, 2, w.dt, w.rescale)
    tbpm.tbpm_get_state(H, ws, 2)
    with pytest.raises(tbpm.TbpmError) as ei:                        # state beyond the call's n_state
        tbpm.tbpm_get_state(H, ws, 3)
    assert ei.value.code == tbpm.TBPM_EINDEX
    other = torch.empty(ws.numel(), dtype=torch.uint8, device=dev)
    with pytest.raises(tbpm.TbpmError) as ei:                        # a workspace this handle never propagated on
        tbpm.tbpm_get_state(H, other, 0)
    assert ei.value.code == tbpm.TBPM_EINVAL


@pytest.mark.parametrize("tau,K", [(0.0, 1), (1e-9, None), (math.pi / 2, 16), (2 * math.pi, 28), (1.0, None), (5.3, None)])
def test_other_time_steps(dev, oracle_mod, tau, K):
    """Different K exercise every flush pattern of the deferred accumulation (1, 2 or 3 pending terms; K = 1, 2)."""
    w = W.make_workload(2, device=dev, Na=40, Nb=36)
    if K is not None:
        assert len(tbpm.tbpm_cheb_coeff(tau)) == K
    run_parity(dev, oracle_mod, w, 2, 7, dt=tau / w.rescale)


def test_prefix_determinism_and_edge_calls(dev, oracle_mod):
    w = W.make_workload(4, device=dev, Lx=64, Ly=64, phi_den=64)
    psi0 = w.psi0(device=dev, n_state=8)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    a, an, _ = tbpm.tbpm_propagate(H, psi0, 12, w.dt, w.rescale)
    b, bn, _ = tbpm.tbpm_propagate(H, psi0, 12, w.dt, w.rescale)
    c, cn, _ = tbpm.tbpm_propagate(H, psi0, 5, w.dt, w.rescale)
    assert torch.equal(a, b) and torch.equal(an, bn)                 # run-to-run bit identical (no float atomics)
    assert torch.equal(a[:, :5], c) and torch.equal(an[:, :5], cn)   # prefix property (reading #7)
    corr, norm2, _ = tbpm.tbpm_propagate(H, psi0, 0, w.dt, w.rescale)  # n_step = 0: success, nothing written
    assert corr.shape == (8, 0)
    corr = torch.full((2, 3), 7.0, dtype=torch.complex128, device=dev)
    tbpm.tbpm_propagate(H, psi0[:0], 3, w.dt, w.rescale, corr=corr)    # n_state = 0: outputs untouched
    assert torch.all(corr == 7.0)
    with pytest.raises(tbpm.TbpmError):
        tbpm.tbpm_propagate(H, psi0, 3, w.dt, -1.0)
    small = torch.empty(1024, dtype=torch.uint8, device=dev)
    with pytest.raises(tbpm.TbpmError) as ei:
        tbpm.tbpm_propagate(H, psi0, 3, w.dt, w.rescale, workspace=small)
    assert ei.value.code == tbpm.TBPM_ENOMEM
    # norm2 = NULL is allowed
    d, dn, _ = tbpm.tbpm_propagate(H, psi0, 5, w.dt, w.rescale, want_norm=False)
    assert dn is None and torch.equal(d, c)


@pytest.mark.parametrize("cfg,over", [(5, dict(L=32)), (4, dict(Lx=128, Ly=32, phi_den=32)), (1, {})])
def test_lattice_and_cluster_kernels_are_deterministic(dev, cfg, over):
    """term_l3, term_sq and k_small_steps: bit-identical reruns and the prefix property (what the parity protocols at scale rest on)."""
    w = W.make_workload(cfg, device=dev, **over)
    n_state = 1 if cfg == 1 else 8
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    a, an, _ = tbpm.tbpm_propagate(H, psi0, 14, w.dt, w.rescale)
    b, bn, _ = tbpm.tbpm_propagate(H, psi0, 14, w.dt, w.rescale)
    c, cn, _ = tbpm.tbpm_propagate(H, psi0, 6, w.dt, w.rescale)
    assert torch.equal(a, b) and torch.equal(an, bn)
    assert torch.equal(a[:, :6], c) and torch.equal(an[:, :6], cn)


def test_windowed_parity_from_snapshot(dev, oracle_mod):
    """Reading/§8(d)(3): download psi at a late step from the GPU, let the oracle advance it and compare the window."""
    w = W.make_workload(2, device=dev, Na=64, Nb=48)
    psi0 = w.psi0(device=dev, n_state=2)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    j, m = 200, 6
    full, _, _ = tbpm.tbpm_propagate(H, psi0, j + m, w.dt, w.rescale)
    _, _, ws = tbpm.tbpm_propagate(H, psi0, j, w.dt, w.rescale)
    snap = torch.stack([tbpm.tbpm_get_state(H, ws, b) for b in range(2)]).cpu().numpy()
    hi, hj, hv, on = to_np(w)
    ref, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0.cpu().numpy(), m, w.dt, w.rescale, psi_start=snap)
    assert np.abs(full[:, j:].cpu().numpy() - ref).max() <= CORR_TOL


# ---------------------------------------------------------------------------------------------------------------------
# a8: LDOS
# ---------------------------------------------------------------------------------------------------------------------
def test_ldos_parity_and_closed_form(dev, oracle_mod):
    w = W.make_workload(5, device=dev, L=14)
    sites = W.ldos_sites(w.n_orb, 11)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    corr, norm2, _ = tbpm.tbpm_ldos(H, sites, 10, w.dt, w.rescale)
    hi, hj, hv, on = to_np(w)
    ref, _ = oracle_mod.ldos(w.n_orb, on, hi, hj, hv, sites.numpy(), 10, w.dt, w.rescale)
    assert np.abs(corr.cpu().numpy() - ref).max() <= CORR_TOL
    assert np.abs(norm2.cpu().numpy() - 1).max() <= NORM_TOL
    with pytest.raises(tbpm.TbpmError):
        tbpm.tbpm_ldos(H, [w.n_orb], 3, w.dt, w.rescale)
    # clean cubic lattice, any L: corr_n = g_n^3 (reading #25) -- needs no oracle
    L, s, nst = 48, 15.0, 40
    n, hi, hj, hv = W.cubic_hops(L, -1.0, dev)
    H = tbpm.tbpm_build(n, None, hi, hj, hv)
    corr, _, _ = tbpm.tbpm_ldos(H, [0, 12345, n - 1], nst, math.pi / s, s)
    q = np.arange(L)
    g = np.exp(-1j * np.outer(np.arange(1, nst + 1), 2 * -1.0 * np.cos(2 * math.pi * q / L)) * math.pi / s).mean(axis=1)
    assert np.abs(corr.cpu().numpy() - g ** 3).max() <= 1e-12


# ---------------------------------------------------------------------------------------------------------------------
# end-to-end host entry
# ---------------------------------------------------------------------------------------------------------------------
def test_corr_host_matches_device_path(dev, oracle_mod):
    w = W.make_workload(2, Na=64, Nb=40)                              # generated on the host
    psi0 = w.psi0(n_state=4).pin_memory()
    n_step = 8
    arena = torch.empty(tbpm.tbpm_corr_host_bytes(w.n_orb, w.n_hop, True, 4, n_step), dtype=torch.uint8, device=dev)
    corr = torch.zeros((4, n_step), dtype=torch.complex128).pin_memory()
    norm2 = torch.zeros((4, n_step), dtype=torch.float64).pin_memory()
    up, down = tbpm.tbpm_corr_host(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val, psi0, n_step, w.dt, w.rescale, arena, corr, norm2)
    assert up == w.n_hop * 24 + w.n_orb * 8 + 4 * w.n_orb * 16 and down == 4 * n_step * 24
    hi, hj, hv, on = to_np(w)
    ref, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0.numpy(), n_step, w.dt, w.rescale)
    assert np.abs(corr.numpy() - ref).max() <= CORR_TOL
    assert np.abs(norm2.numpy() - 1).max() <= NORM_TOL


# ---------------------------------------------------------------------------------------------------------------------
# full-size configs, in the launch configuration bench.py times
# ---------------------------------------------------------------------------------------------------------------------
def load_golden(cfg, state):
    """tests/golden/corr_full_cfg<cfg>_state<state>.txt: a full-length ORACLE run written by tests/golden/make_full_length.py
    (which calls only oracle/): columns step, Re corr, Im corr, norm2."""
    path = os.path.join(os.path.dirname(__file__), "golden", f"corr_full_cfg{cfg}_state{state}.txt")
    if not os.path.exists(path):
        return None
    a = np.loadtxt(path)
    return a[:, 1] + 1j * a[:, 2], a[:, 3]


def test_config2_full_length(dev):
    """BASELINE.json:configs[1] exactly: 4 states x 1024 steps at 2,097,152 orbitals, EVERY entry of corr against the cached
    full-length oracle run (parity protocols (1) and (6) of SURVEY 8(d))."""
    w = W.make_workload(2, device=dev)
    psi0 = w.psi0(device=dev)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    corr, norm2, _ = tbpm.tbpm_propagate(H, psi0, w.n_step, w.dt, w.rescale)
    torch.cuda.synchronize()
    corr, norm2 = corr.cpu().numpy(), norm2.cpu().numpy()
    for b in range(4):
        ref, refn = load_golden(2, b)
        assert ref.shape == (w.n_step,)
        assert np.abs(corr[b] - ref).max() <= CORR_TOL
        assert np.abs(norm2[b] - refn).max() <= NORM_TOL
    assert np.abs(norm2 - 1).max() <= NORM_TOL


def test_dos_from_corr(dev, oracle_mod):
    """NEXT-1 (tbpm_dos): Hann-windowed direct transform of the state-averaged correlation against the oracle's
    dos_from_corr (itself pinned by the honeycomb and chain closed forms, tests/test_oracle_pins.py)."""
    w = W.make_workload(2, device=dev, Na=48, Nb=40, n_state=3)
    psi0 = w.psi0(n_state=3)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    n_step = 200
    corr, _, _ = tbpm.tbpm_propagate(H, psi0, n_step, w.dt, w.rescale)
    E, D = tbpm.tbpm_dos(corr, w.dt, w.rescale)
    torch.cuda.synchronize()
    Eo, Do = oracle_mod.dos_from_corr(corr.cpu().numpy().mean(axis=0), w.rescale)
    assert E.shape == (2 * n_step + 1,)
    assert np.abs(E.cpu().numpy() - Eo).max() <= 1e-12 * w.rescale
    assert np.abs(D.cpu().numpy() - Do).max() <= 1e-10 * np.abs(Do).max()
    assert abs(float(D.sum()) * w.rescale / n_step - 1.0) < 2e-2           # integrates to one state per orbital
    E1, D1 = tbpm.tbpm_dos(corr[1], w.dt, w.rescale)                      # one state, 1-D input
    _, D1o = oracle_mod.dos_from_corr(corr[1].cpu().numpy(), w.rescale)
    assert np.abs(D1.cpu().numpy() - D1o).max() <= 1e-10 * np.abs(D1o).max()
    assert tbpm.lib().tbpm_dos(None, 1, 4, 0.1, 1.0, None, None, None) == tbpm.TBPM_EINVAL


FULL = os.environ.get("TBPM_TEST_FULL", "1") != "0"


def eigen_check(dev, w, psi, E, n_step):
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    corr, norm2, _ = tbpm.tbpm_propagate(H, psi[None, :].contiguous(), n_step, w.dt, w.rescale)
    n = np.arange(1, n_step + 1)
    assert np.abs(corr.cpu().numpy()[0] - np.exp(-1j * n * math.pi * E / w.rescale)).max() <= CORR_TOL
    assert np.abs(norm2.cpu().numpy() - 1).max() <= NORM_TOL


@pytest.mark.skipif(not FULL, reason="TBPM_TEST_FULL=0")
def test_full_size_closed_form_eigenstates(dev):
    """Reading #10: uniform / staggered states are exact eigenstates of the clean periodic lattices, so
    corr_n = exp(-i n tau E/s) and norm2 = 1 at 16-33 M orbitals with no oracle at all."""
    w = W.make_workload(3, device=dev, vac=0.0)                       # clean honeycomb 4096x4096, 33.5 M orbitals
    N = w.n_orb
    eigen_check(dev, w, torch.full((N,), 1 / math.sqrt(N), dtype=torch.complex128, device=dev), 3 * -2.7, 24)
    stag = torch.where(torch.arange(N, device=dev) % 2 == 0, 1.0, -1.0).to(torch.complex128) / math.sqrt(N)
    eigen_check(dev, w, stag, -3 * -2.7, 24)
    del w, stag
    n, hi, hj, hv = W.cubic_hops(256, -1.0, dev)                      # clean cubic 256^3
    w = W.Workload("cubic-clean", n, hi, hj, hv, None, 1, 1, 15.0)
    eigen_check(dev, w, torch.full((n,), 1 / math.sqrt(n), dtype=torch.complex128, device=dev), -6.0, 24)


# states compared with the oracle at full size: one from EVERY tile of 8 (config 5: tiles 0-3; its LDOS leg: one site of each of the 8 tiles)
FULL_SAMPLE = {2: [0, 3], 3: [0], 4: [1, 6], 5: [2, 13, 17, 30]}
LDOS_SAMPLE = [0, 9, 18, 27, 36, 45, 54, 63]
FULL_GOLDEN_STATE = {3: 0, 4: 3, 5: 5}          # tests/golden/make_full_length.py: STATES


@pytest.mark.skipif(not FULL, reason="TBPM_TEST_FULL=0")
@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_full_size_prefix_parity(dev, oracle_mod, cfg):
    """Configs 2-5 at BASELINE.json's full size with all their states batched as bench.py runs them (same kernels, same tile
    order).  Protocol (2) of SURVEY 8(d): the first m = 16 steps of a state from every tile against the oracle (OpenMP row form);
    the norm of every state at every step; and, at full size, the exported CSR against the oracle's builder bit for bit."""
    m = 16
    w = W.make_workload(cfg, device=dev)
    psi0 = w.psi0(device=dev)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    assert H.nnz == w.nnz
    corr, norm2, _ = tbpm.tbpm_propagate(H, psi0, m, w.dt, w.rescale)
    torch.cuda.synchronize()
    assert np.abs(norm2.cpu().numpy() - 1).max() <= NORM_TOL
    hi, hj, hv, on = to_np(w)
    sample = FULL_SAMPLE[cfg]
    ref, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0[sample].cpu().numpy(), m, w.dt, w.rescale, form="csr")
    assert np.abs(corr[sample].cpu().numpy() - ref).max() <= CORR_TOL
    if cfg == 3:
        assert abs(w.n_orb - 30198989) < 20000 and H.max_row_nnz == 3
    if cfg in (3, 4):                                                 # canonical CSR at full size, bit for bit
        del psi0, corr, norm2
        assert_csr_bit_exact(H, oracle_mod, w)
    if cfg == 5:                                                      # LDOS leg of config 5 on the same H: 64 sites = 8 tiles
        sites = w.sites()
        lc, ln, _ = tbpm.tbpm_ldos(H, sites, 8, w.dt, w.rescale)
        lref, _ = oracle_mod.ldos(w.n_orb, on, hi, hj, hv, sites[LDOS_SAMPLE].numpy(), 8, w.dt, w.rescale, form="csr")
        assert np.abs(lc[LDOS_SAMPLE].cpu().numpy() - lref).max() <= CORR_TOL
        assert np.abs(ln.cpu().numpy() - 1).max() <= NORM_TOL


@pytest.mark.skipif(not FULL, reason="TBPM_TEST_FULL=0")
@pytest.mark.parametrize("cfg,j", [(3, 200), (4, 200), (5, 120)])
def test_full_size_windowed_parity(dev, oracle_mod, cfg, j):
    """Protocol (3) of SURVEY 8(d) at full size: psi at a late step j is downloaded from the GPU with tbpm_get_state, the oracle
    advances it m = 4 steps and must reproduce corr[:, j : j + m] of a longer GPU run; protocol (4): |norm2 - 1| <= 1e-12 at
    every one of the j + m steps for every state."""
    m = 4
    w = W.make_workload(cfg, device=dev)
    psi0 = w.psi0(device=dev)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    ws = torch.empty(tbpm.tbpm_propagate_bytes(H, w.n_state), dtype=torch.uint8, device=dev)
    full, norm2, _ = tbpm.tbpm_propagate(H, psi0, j + m, w.dt, w.rescale, workspace=ws)
    full = full.clone()
    assert np.abs(norm2.cpu().numpy() - 1).max() <= NORM_TOL
    head, _, _ = tbpm.tbpm_propagate(H, psi0, j, w.dt, w.rescale, workspace=ws)
    assert torch.equal(head, full[:, :j])                            # prefix property, bit for bit
    sample = FULL_SAMPLE[cfg][-2:]
    snap = torch.stack([tbpm.tbpm_get_state(H, ws, b) for b in sample]).cpu().numpy()
    hi, hj, hv, on = to_np(w)
    ref, _ = oracle_mod.propagate(w.n_orb, on, hi, hj, hv, psi0[sample].cpu().numpy(), m, w.dt, w.rescale, psi_start=snap, form="csr")
    assert np.abs(full[sample][:, j:].cpu().numpy() - ref).max() <= CORR_TOL


@pytest.mark.skipif(not FULL, reason="TBPM_TEST_FULL=0")
@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_length_against_cached_oracle(dev, cfg):
    """Protocol (6) of SURVEY 8(d): a FULL-LENGTH GPU run (1024 / 2048 / 1024 steps) of the tile that holds the state whose
    full-length oracle run is cached under tests/golden/ (tests/golden/make_full_length.py, oracle only), every entry of that
    state's corr <= 1e-10, and |norm2 - 1| <= 1e-12 at every step for every state of the tile (protocol (4))."""
    state = FULL_GOLDEN_STATE[cfg]
    gold = load_golden(cfg, state)
    if gold is None:
        pytest.skip(f"tests/golden/corr_full_cfg{cfg}_state{state}.txt has not been generated")
    ref, refn = gold
    w = W.make_workload(cfg, device=dev)
    n_state = min(w.n_state, 8)                                       # tile 0 of the batch: bit-identical to the full batch's tile 0
    psi0 = w.psi0(device=dev, n_state=n_state)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val)
    corr, norm2, _ = tbpm.tbpm_propagate(H, psi0, w.n_step, w.dt, w.rescale)
    torch.cuda.synchronize()
    assert ref.shape == (w.n_step,)
    err = np.abs(corr[state].cpu().numpy() - ref).max()
    print(f"config {cfg} full length: max|dcorr| = {err:.3e}, max|norm2 - 1| = {np.abs(norm2.cpu().numpy() - 1).max():.3e}")
    assert err <= CORR_TOL
    assert np.abs(norm2[state].cpu().numpy() - refn).max() <= NORM_TOL
    assert np.abs(norm2.cpu().numpy() - 1).max() <= NORM_TOL
