"""Pins of the seeded input generators (structure of the synthetic workloads)."""
import math

import numpy as np
import pytest
import torch

from paper_2509_26309_b200 import workloads as W


def test_counter_hash_is_reproducible_and_uniform():
    key = W.stream_key(W.MASTER_SEED, W.STREAM_PSI0, 3)
    u = W.counter_uniform(key, 0, 200000)
    v = W.counter_uniform(key, 1000, 50)
    assert torch.equal(u[1000:1050], v)                              # counter based: any window can be regenerated
    assert 0.0 <= float(u.min()) and float(u.max()) < 1.0
    assert float(u.mean()) == pytest.approx(0.5, abs=3e-3)
    assert float(u.var()) == pytest.approx(1 / 12, abs=2e-3)
    # host reference of the same mixer on python ints
    z = (key + 1 * 0x9E3779B97F4A7C15) & ((1 << 64) - 1)
    assert float(u[0]) == (W._mix64_i(z) >> 11) / 2 ** 53


def test_random_phase_state():
    p = W.random_phase_states(4096, 3)
    assert p.dtype == torch.complex128 and p.shape == (3, 4096)
    assert torch.allclose(p.abs(), torch.full((3, 4096), 1 / 64.0, dtype=torch.float64), atol=1e-15)
    assert float((p.abs() ** 2).sum(1).sub(1).abs().max()) < 1e-13   # pin #12
    assert abs(complex(torch.vdot(p[0], p[1]))) < 0.1                 # different sub-streams are uncorrelated


def test_honeycomb_structure():
    n, hi, hj, hv = W.honeycomb_hops(5, 7)
    assert n == 70 and hi.numel() == 3 * 35
    deg = torch.bincount(torch.cat([hi, hj]).long(), minlength=n)
    assert torch.all(deg == 3)                                        # every row has exactly 3 entries
    assert torch.all((hi % 2) != (hj % 2))                            # bipartite A-B only
    pairs = {(min(a, b), max(a, b)) for a, b in zip(hi.tolist(), hj.tolist())}
    assert len(pairs) == hi.numel()                                   # each pair once
    # PAPER.md:762-764 connectivity for cell (1,2): A=(1*7+2)*2=18
    assert (18, 19) in pairs and (19, ((2 * 7 + 2) * 2)) in pairs and (19, (1 * 7 + 3) * 2) in pairs
    assert torch.all(hv == complex(-2.7, 0))


def test_vacancies():
    n, hi, hj, hv = W.honeycomb_hops(256, 256)
    n2, hi2, hj2, hv2, keep = W.apply_vacancies(n, hi, hj, hv, 0.10)
    assert n2 == int(keep.sum()) and n2 / n == pytest.approx(0.90, abs=3e-3)
    assert int(hi2.max()) < n2 and int(hj2.max()) < n2
    deg = torch.bincount(torch.cat([hi2, hj2]).long(), minlength=n2)
    hist = torch.bincount(deg, minlength=4).double() / n2
    expect = [math.comb(3, k) * 0.9 ** k * 0.1 ** (3 - k) for k in range(4)]   # Binomial(3, 0.9)
    assert np.allclose(hist.numpy(), expect, atol=4e-3)
    assert int((deg == 0).sum()) > 0                                  # isolated survivors are kept (no trim)


def test_peierls_flux_invariants():
    Lx, Ly, den = 16, 8, 16
    n, hi, hj, hv = W.square_peierls_hops(Lx, Ly, -1.0, 0.2, 1, den)
    H = {}
    for i, j, v in zip(hi.tolist(), hj.tolist(), hv.tolist()):
        H[(i, j)] = v
        H[(j, i)] = v.conjugate()
    assert len(H) == 2 * hi.numel()                                   # no duplicates
    phi = 1 / den
    idx = lambda x, y: (y % Ly) * Lx + (x % Lx)
    hop = lambda a, b: H[(b, a)]                                      # amplitude for the move a -> b is <b|H|a>
    for x in range(Lx):
        for y in range(Ly):
            a, b, c, d = idx(x, y), idx(x + 1, y), idx(x + 1, y + 1), idx(x, y + 1)
            loop = hop(a, b) * hop(b, c) * hop(c, d) * hop(d, a)      # counter-clockwise plaquette, t^4 = 1
            assert loop == pytest.approx(np.exp(2j * math.pi * phi), abs=1e-12)
            tri = hop(a, b) * hop(b, c) * hop(c, a)                   # NN-NN-NNN triangle = half a plaquette
            assert tri / abs(tri) == pytest.approx(np.exp(1j * math.pi * phi), abs=1e-12)
    rowsum = np.zeros(n)
    for (i, j), v in H.items():
        rowsum[i] += abs(v)
    assert np.allclose(rowsum, 4.8)                                   # Gershgorin bound = s exactly (reading #18)
    with pytest.raises(ValueError):
        W.square_peierls_hops(10, 8, -1.0, 0.2, 1, 16)                # phi*Lx not an integer


def test_cubic_and_anderson_and_sites():
    n, hi, hj, hv = W.cubic_hops(5)
    deg = torch.bincount(torch.cat([hi, hj]).long(), minlength=n)
    assert n == 125 and torch.all(deg == 6)
    on = W.anderson_onsite(100000, 16.5)
    assert float(on.min()) >= -8.25 and float(on.max()) < 8.25
    assert float(on.mean()) == pytest.approx(0, abs=0.08) and float(on.var()) == pytest.approx(16.5 ** 2 / 12, rel=0.02)
    s = W.ldos_sites(1000, 64)
    assert len(set(s.tolist())) == 64 and int(s.max()) < 1000
    assert torch.equal(s, W.ldos_sites(1000, 64))


def test_config_shapes_match_baseline_json():
    w = W.make_workload(1)
    assert (w.n_orb, w.nnz, w.n_state, w.n_step, w.rescale) == (8192, 24576, 1, 256, 9.0)
    assert w.rescale * w.dt == pytest.approx(math.pi)
    for cfg, n_orb, n_state, n_step, s in ((2, 2097152, 4, 1024, 9.5), (3, None, 1, 1024, 9.0), (4, 16777216, 8, 2048, 4.8),
                                           (5, 16777216, 32, 1024, 15.0)):
        p = W._FULL[cfg]
        assert (p["n_state"], p["n_step"], p["rescale"]) == (n_state, n_step, s)
    assert W._FULL[5]["ldos"] == 64
