"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/tbpm.h declares, and its host logic
(coefficients, sizes, argument checks) is right.  No compute call is made without a GPU."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest
import scipy.special as sp

from paper_2509_26309_b200 import tbpm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tbpm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tbpm_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_symbols()
    assert {"tbpm_build", "tbpm_propagate", "tbpm_ldos", "tbpm_export_csr", "tbpm_get_state", "tbpm_cheb_coeff",
            "tbpm_corr_host"} <= set(names)
    L = tbpm.lib()
    for n in names:
        assert hasattr(L, n), n
    assert "sm_100a" in tbpm.tbpm_version()


def test_built_for_sm_100a():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", tbpm._build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_cheb_coeff_host_logic():
    for tau, K in ((math.pi, 21), (math.pi / 2, 16), (2 * math.pi, 28), (0.0, 1)):
        c = tbpm.tbpm_cheb_coeff(tau).numpy()
        assert len(c) == K
        J = sp.jv(np.arange(K), tau)
        ref = np.where(np.arange(K) == 0, 1, 2) * (-1j) ** np.arange(K) * J
        assert np.abs(c - ref).max() < 5e-16
    for tau in (0.3, 7.7, 40.0, 300.0):
        c = tbpm.tbpm_cheb_coeff(tau).numpy()
        x = np.linspace(-1, 1, 101)
        Tk = np.cos(np.outer(np.arange(len(c)), np.arccos(x)))
        assert np.abs(c @ Tk - np.exp(-1j * tau * x)).max() < 2e-14 * max(1.0, tau)     # Jacobi-Anger
    K = C.c_int(0)
    buf = (C.c_double * 8)()
    assert tbpm.lib().tbpm_cheb_coeff(math.pi, 1e-15, 4, C.byref(K), buf) == tbpm.TBPM_ENOMEM and K.value == 21
    assert tbpm.lib().tbpm_cheb_coeff(-1.0, 1e-15, 4, C.byref(K), buf) == tbpm.TBPM_EINVAL


def test_fermi_coeff_host_logic():
    """NEXT-4: sum_k c_k T_k(x) = 1 / (exp(beta (s x - mu)) + 1) on [-1, 1] (closed form), the complement, beta = 0, bad arguments."""
    for beta, mu, s in ((2.0, 0.3, 4.8), (11.0, -1.0, 4.8), (0.5, 0.0, 9.0)):
        c = tbpm.tbpm_fermi_coeff(beta, mu, s).numpy()
        g = tbpm.tbpm_fermi_coeff(beta, mu, s, one_minus=True).numpy()
        x = np.linspace(-1, 1, 201)
        Tk = np.cos(np.outer(np.arange(len(c)), np.arccos(x)))
        f = 1.0 / (np.exp(beta * (s * x - mu)) + 1.0)
        assert np.abs(c @ Tk - f).max() < 1e-11 and np.abs(g @ Tk - (1 - f)).max() < 1e-11
        assert abs(c[-1]) >= 1e-13
    assert tbpm.tbpm_fermi_coeff(0.0, 0.0, 3.0).tolist() == [0.5]
    K = C.c_int(0)
    buf = (C.c_double * 8)()
    L = tbpm.lib()
    assert L.tbpm_fermi_coeff(11.0, 0.0, 4.8, 0, 1e-13, 4, C.byref(K), buf) == tbpm.TBPM_ENOMEM and K.value > 4
    assert L.tbpm_fermi_coeff(-1.0, 0.0, 4.8, 0, 1e-13, 4, C.byref(K), buf) == tbpm.TBPM_EINVAL
    assert L.tbpm_corr_ac(None, None, None, None, 1, 1, 0.1, 1.0, 1.0, 0.0, None, None, 0, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_haydock(None, None, 1, 1, None, None, None, 0, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_propagate_qe(None, None, 1, 1, 0.1, 1.0, None, 0, None, None, None, None, 0, None) == tbpm.TBPM_EINVAL


def test_sizes_and_argument_checks():
    p, s = tbpm.tbpm_build_bytes(8192, 12288, False)
    assert p >= 24576 * 20 + 8193 * 8 and s > 0
    p2, _ = tbpm.tbpm_build_bytes(8192, 12288, True)
    assert p2 > p
    with pytest.raises(tbpm.TbpmError):
        tbpm.tbpm_build_bytes(1 << 31, 10, False)
    with pytest.raises(tbpm.TbpmError):
        tbpm.tbpm_build_bytes(10, 1 << 31, False)                    # nnz would not fit 32-bit row offsets
    L = tbpm.lib()
    assert L.tbpm_propagate(None, None, 1, 1, 0.1, 1.0, None, None, None, 0, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_ldos(None, None, 1, 1, 0.1, 1.0, None, None, None, 0, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_get_state(None, None, 0, None, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_export_csr(None, None, None, None, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_check_bound(None, 1.0) == tbpm.TBPM_EINVAL
    assert L.tbpm_dos(None, 1, 4, 0.1, 1.0, None, None, None) == tbpm.TBPM_EINVAL
    assert L.tbpm_dos(None, 0, 4, 0.1, 1.0, None, None, None) == tbpm.TBPM_OK        # nothing to do
    assert L.tbpm_dos(None, 1, 4, 0.1, -1.0, None, None, None) == tbpm.TBPM_EINVAL
    b = tbpm.tbpm_corr_host_bytes(8192, 12288, False, 1, 256)
    assert b > p
    for code in range(0, -8, -1):
        assert tbpm.tbpm_strerror(code) != "unknown error code"
    assert tbpm.tbpm_strerror(-99) == "unknown error code"


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    hi = torch.zeros(3, dtype=torch.int32)
    with pytest.raises(tbpm.TbpmError):                              # host tensors are refused: there is no CPU path
        tbpm.tbpm_build(4, None, hi, hi, torch.zeros(3, dtype=torch.complex128))
