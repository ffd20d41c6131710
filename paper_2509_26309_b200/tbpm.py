"""Thin Python binding of libtbpm.so (include/tbpm.h): argument marshalling only.

Function names mirror the C ABI.  torch is used for device memory and streams only; every step of the path runs in
the library's CUDA kernels.  There is no CPU fallback: if the library is missing or no CUDA device is usable, the
calls raise.  Nothing here imports `oracle/`.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import torch

from . import build as _build

TBPM_VALIDATE, TBPM_HOPS_FULL, TBPM_NO_TABLE = 1, 2, 4
TBPM_OPT_TILE, TBPM_OPT_KERNEL = 1, 2
TBPM_LATTICE_CUBIC, TBPM_LATTICE_SQUARE8, TBPM_LATTICE_NEAR16 = 2, 3, 4
TBPM_OK, TBPM_EINVAL, TBPM_EINDEX, TBPM_EDIAG, TBPM_EDUP, TBPM_ENOMEM, TBPM_ECUDA, TBPM_EBOUND = 0, -1, -2, -3, -4, -5, -6, -7
TBPM_ETOOBIG = -8
TBPM_STATIC_WORKSPACE_BYTES = 8 << 20

_lib = None


class TbpmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {tbpm_strerror(code)} (code {code})")


def lib() -> C.CDLL:
    """Load libtbpm.so (built in-tree by paper_2509_26309_b200/build.py).  Raises if it cannot be loaded."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if not os.path.exists(path):
            path = _build.build()
        L = C.CDLL(path)
        vp, i64, i32, u32, dbl, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_uint32, C.c_double, C.c_size_t
        P = C.POINTER
        L.tbpm_strerror.restype = C.c_char_p
        L.tbpm_strerror.argtypes = [C.c_int]
        L.tbpm_version.restype = C.c_char_p
        L.tbpm_cheb_coeff.argtypes = [dbl, dbl, C.c_int, P(C.c_int), vp]
        L.tbpm_build_bytes.argtypes = [i64, i64, C.c_int, u32, P(sz), P(sz)]
        L.tbpm_build.argtypes = [i64, vp, i64, vp, vp, vp, u32, vp, sz, vp, sz, vp, P(vp)]
        L.tbpm_ham_info.argtypes = [vp, P(i64), P(i64), P(i32), P(sz), P(i32), P(dbl)]
        L.tbpm_check_bound.argtypes = [vp, dbl]
        L.tbpm_ham_lattice_info.argtypes = [vp, P(i32), P(sz)]
        L.tbpm_export_csr.argtypes = [vp, vp, vp, vp, vp]
        L.tbpm_free.argtypes = [vp]
        L.tbpm_free.restype = None
        L.tbpm_propagate_bytes.argtypes = [vp, C.c_int, P(sz)]
        L.tbpm_propagate.argtypes = [vp, vp, C.c_int, C.c_int, dbl, dbl, vp, vp, vp, sz, vp]
        L.tbpm_propagate_static.argtypes = [vp, vp, C.c_int, C.c_int, dbl, dbl, vp, vp, vp]
        L.tbpm_ldos.argtypes = [vp, vp, C.c_int, C.c_int, dbl, dbl, vp, vp, vp, sz, vp]
        L.tbpm_get_state.argtypes = [vp, vp, C.c_int, vp, vp]
        L.tbpm_dos.argtypes = [vp, C.c_int, C.c_int, dbl, dbl, vp, vp, vp]
        L.tbpm_propagate_qe_bytes.argtypes = [vp, C.c_int, C.c_int, P(sz)]
        L.tbpm_propagate_qe.argtypes = [vp, vp, C.c_int, C.c_int, dbl, dbl, vp, C.c_int, vp, vp, vp, vp, sz, vp]
        L.tbpm_haydock.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp, vp, sz, vp]
        L.tbpm_fermi_coeff.argtypes = [dbl, dbl, dbl, C.c_int, dbl, C.c_int, P(C.c_int), vp]
        L.tbpm_corr_ac_bytes.argtypes = [vp, C.c_int, P(sz)]
        L.tbpm_corr_ac.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, dbl, dbl, dbl, dbl, vp, vp, sz, vp]
        L.tbpm_corr_dp.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, dbl, dbl, dbl, dbl, vp, vp, sz, vp]
        L.tbpm_haydock_ldos.argtypes = [vp, vp, C.c_int, C.c_int, vp, C.c_int, dbl, vp, vp]
        L.tbpm_last_launch_count.restype = i64
        L.tbpm_last_launch_count.argtypes = [vp]
        L.tbpm_set_option.argtypes = [vp, C.c_int, i64]
        L.tbpm_total_launch_count.restype = i64
        L.tbpm_corr_host_bytes.argtypes = [i64, i64, C.c_int, C.c_int, C.c_int, u32, P(sz)]
        L.tbpm_corr_host.argtypes = [i64, vp, i64, vp, vp, vp, u32, vp, C.c_int, C.c_int, dbl, dbl, vp, vp, vp, sz, vp, P(sz), P(sz)]
        _lib = L
    return _lib


def _check(rc: int, where: str):
    if rc != TBPM_OK:
        raise TbpmError(rc, where)


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(device) -> C.c_void_p:
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _need_cuda(*tensors):
    for t in tensors:
        if t is not None and not t.is_cuda:
            raise TbpmError(TBPM_ECUDA, "tbpm: device tensors required (there is no CPU path)")


def _bytes(n: int, device) -> torch.Tensor:
    """Caller-owned raw device buffer (256-byte aligned by the torch caching allocator)."""
    return torch.empty(max(int(n), 256), dtype=torch.uint8, device=device)


def tbpm_strerror(code: int) -> str:
    return lib().tbpm_strerror(code).decode()


def tbpm_version() -> str:
    return lib().tbpm_version().decode()


def tbpm_cheb_coeff(tau: float, tol: float = 1e-15, kcap: int = 8192) -> torch.Tensor:
    """Host only: complex128 [K] Chebyshev coefficients c_k = (2-delta_k0)(-i)^k J_k(tau)."""
    buf = torch.empty(kcap, dtype=torch.complex128)
    K = C.c_int(0)
    _check(lib().tbpm_cheb_coeff(tau, tol, kcap, C.byref(K), C.c_void_p(buf.data_ptr())), "tbpm_cheb_coeff")
    return buf[: K.value].clone()


def tbpm_build_bytes(n_orb: int, n_hop: int, has_onsite: bool, flags: int = 0) -> Tuple[int, int]:
    p, s = C.c_size_t(0), C.c_size_t(0)
    _check(lib().tbpm_build_bytes(n_orb, n_hop, int(has_onsite), flags, C.byref(p), C.byref(s)), "tbpm_build_bytes")
    return p.value, s.value


class Hamiltonian:
    """Owner of the opaque tbpm_ham handle and of the `persist` device buffer it points into."""

    def __init__(self, handle: int, persist: torch.Tensor, device):
        self.handle = C.c_void_p(handle)
        self.persist = persist
        self.device = device
        n, nnz, mr, mb, nt, g = C.c_int64(0), C.c_int64(0), C.c_int32(0), C.c_size_t(0), C.c_int32(0), C.c_double(0)
        _check(lib().tbpm_ham_info(self.handle, C.byref(n), C.byref(nnz), C.byref(mr), C.byref(mb), C.byref(nt), C.byref(g)), "tbpm_ham_info")
        self.n_orb, self.nnz, self.max_row_nnz = n.value, nnz.value, mr.value
        self.matrix_bytes_per_term, self.n_table, self.gershgorin = mb.value, nt.value, g.value
        kind, lb = C.c_int32(0), C.c_size_t(0)
        _check(lib().tbpm_ham_lattice_info(self.handle, C.byref(kind), C.byref(lb)), "tbpm_ham_lattice_info")
        self.lattice_kind, self.lattice_bytes_per_term = kind.value, lb.value

    def __del__(self):
        try:
            if self.handle:
                lib().tbpm_free(self.handle)
                self.handle = None
        except Exception:
            pass


def tbpm_build(n_orb: int, onsite: Optional[torch.Tensor], hop_i: torch.Tensor, hop_j: torch.Tensor, hop_val: torch.Tensor,
               flags: int = 0) -> Hamiltonian:
    """hop_i/hop_j int32 [n_hop], hop_val complex128 [n_hop], onsite float64 [n_orb] or None; all on one CUDA device."""
    _need_cuda(hop_i, hop_j, hop_val, onsite)
    dev = hop_i.device
    assert hop_i.dtype == torch.int32 and hop_j.dtype == torch.int32 and hop_val.dtype == torch.complex128
    assert onsite is None or (onsite.dtype == torch.float64 and onsite.numel() == n_orb)
    hop_i, hop_j, hop_val = hop_i.contiguous(), hop_j.contiguous(), hop_val.contiguous()
    onsite = None if onsite is None else onsite.contiguous()
    n_hop = hop_i.numel()
    pb, sb = tbpm_build_bytes(n_orb, n_hop, onsite is not None, flags)
    persist, scratch = _bytes(pb, dev), _bytes(sb, dev)
    out = C.c_void_p(0)
    with torch.cuda.device(dev):
        rc = lib().tbpm_build(n_orb, _ptr(onsite), n_hop, _ptr(hop_i), _ptr(hop_j), _ptr(hop_val), flags, _ptr(persist), pb,
                              _ptr(scratch), sb, _stream(dev), C.byref(out))
    _check(rc, "tbpm_build")
    return Hamiltonian(out.value, persist, dev)


def tbpm_check_bound(H: Hamiltonian, rescale: float) -> int:
    return lib().tbpm_check_bound(H.handle, rescale)


def tbpm_export_csr(H: Hamiltonian):
    """Canonical CSR as device tensors (rowptr int64 [n_orb+1], col int32 [nnz], val complex128 [nnz])."""
    dev = H.device
    rowptr = torch.empty(H.n_orb + 1, dtype=torch.int64, device=dev)
    col = torch.empty(max(H.nnz, 1), dtype=torch.int32, device=dev)
    val = torch.empty(max(H.nnz, 1), dtype=torch.complex128, device=dev)
    with torch.cuda.device(dev):
        _check(lib().tbpm_export_csr(H.handle, _ptr(rowptr), _ptr(col), _ptr(val), _stream(dev)), "tbpm_export_csr")
    return rowptr, col[: H.nnz], val[: H.nnz]


def tbpm_propagate_bytes(H: Hamiltonian, n_state: int) -> int:
    b = C.c_size_t(0)
    _check(lib().tbpm_propagate_bytes(H.handle, n_state, C.byref(b)), "tbpm_propagate_bytes")
    return b.value


def tbpm_propagate(H: Hamiltonian, psi0: torch.Tensor, n_step: int, dt: float, rescale: float, workspace: Optional[torch.Tensor] = None,
                   want_norm: bool = True, corr: Optional[torch.Tensor] = None, norm2: Optional[torch.Tensor] = None):
    """psi0 complex128 [n_state][n_orb] on the device -> (corr complex128 [n_state][n_step], norm2 float64 or None, workspace)."""
    _need_cuda(psi0)
    dev = H.device
    assert psi0.dtype == torch.complex128 and psi0.dim() == 2 and psi0.shape[1] == H.n_orb
    psi0 = psi0.resolve_conj().contiguous()
    n_state = psi0.shape[0]
    wb = tbpm_propagate_bytes(H, n_state)
    if workspace is None:
        workspace = _bytes(wb, dev)
    if corr is None:
        corr = torch.zeros((n_state, n_step), dtype=torch.complex128, device=dev)
    if norm2 is None and want_norm:
        norm2 = torch.zeros((n_state, n_step), dtype=torch.float64, device=dev)
    with torch.cuda.device(dev):
        rc = lib().tbpm_propagate(H.handle, _ptr(psi0), n_state, n_step, dt, rescale, _ptr(corr), _ptr(norm2), _ptr(workspace),
                                  workspace.numel(), _stream(dev))
    _check(rc, "tbpm_propagate")
    return corr, norm2, workspace


def tbpm_propagate_static(H: Hamiltonian, psi0: torch.Tensor, n_step: int, dt: float, rescale: float, corr: Optional[torch.Tensor] = None,
                          norm2: Optional[torch.Tensor] = None, want_norm: bool = True):
    """tbpm_propagate without a workspace: the library's static device array serves (small models only, TbpmError(TBPM_ETOOBIG)
    beyond TBPM_STATIC_WORKSPACE_BYTES).  The C call allocates nothing; pass `corr` / `norm2` to keep this wrapper from allocating too.
    Returns (corr, norm2)."""
    _need_cuda(psi0)
    dev = H.device
    assert psi0.dtype == torch.complex128 and psi0.dim() == 2 and psi0.shape[1] == H.n_orb
    psi0 = psi0.resolve_conj().contiguous()
    n_state = psi0.shape[0]
    if corr is None:
        corr = torch.zeros((n_state, n_step), dtype=torch.complex128, device=dev)
    if norm2 is None and want_norm:
        norm2 = torch.zeros((n_state, n_step), dtype=torch.float64, device=dev)
    with torch.cuda.device(dev):
        rc = lib().tbpm_propagate_static(H.handle, _ptr(psi0), n_state, n_step, dt, rescale, _ptr(corr), _ptr(norm2), _stream(dev))
    _check(rc, "tbpm_propagate_static")
    return corr, norm2


def tbpm_ldos(H: Hamiltonian, sites, n_step: int, dt: float, rescale: float, workspace: Optional[torch.Tensor] = None,
              want_norm: bool = True):
    """sites: host int64 [n_site] -> (corr complex128 [n_site][n_step], norm2, workspace)."""
    dev = H.device
    sites = torch.as_tensor(sites, dtype=torch.int64, device="cpu").contiguous()
    n_site = sites.numel()
    wb = tbpm_propagate_bytes(H, n_site)
    if workspace is None:
        workspace = _bytes(wb, dev)
    corr = torch.zeros((n_site, n_step), dtype=torch.complex128, device=dev)
    norm2 = torch.zeros((n_site, n_step), dtype=torch.float64, device=dev) if want_norm else None
    with torch.cuda.device(dev):
        rc = lib().tbpm_ldos(H.handle, C.c_void_p(sites.data_ptr()), n_site, n_step, dt, rescale, _ptr(corr), _ptr(norm2),
                             _ptr(workspace), workspace.numel(), _stream(dev))
    _check(rc, "tbpm_ldos")
    return corr, norm2, workspace


def tbpm_propagate_qe(H: Hamiltonian, psi0: torch.Tensor, energies, n_step: int, dt: float, rescale: float):
    """NEXT-3: (corr, norm2, qe complex128 [n_state][n_energy][n_orb]) for host energies [n_energy]."""
    _need_cuda(psi0)
    dev = H.device
    psi0 = psi0.contiguous()
    n_state = psi0.shape[0]
    en = torch.as_tensor(energies, dtype=torch.float64, device="cpu").contiguous()
    n_e = en.numel()
    wb = C.c_size_t(0)
    _check(lib().tbpm_propagate_qe_bytes(H.handle, n_state, n_e, C.byref(wb)), "tbpm_propagate_qe_bytes")
    ws = _bytes(wb.value, dev)
    corr = torch.zeros((n_state, n_step), dtype=torch.complex128, device=dev)
    norm2 = torch.zeros((n_state, n_step), dtype=torch.float64, device=dev)
    qe = torch.zeros((n_state, n_e, H.n_orb), dtype=torch.complex128, device=dev)
    with torch.cuda.device(dev):
        rc = lib().tbpm_propagate_qe(H.handle, _ptr(psi0), n_state, n_step, dt, rescale, C.c_void_p(en.data_ptr()), n_e, _ptr(corr),
                                     _ptr(norm2), _ptr(qe), _ptr(ws), ws.numel(), _stream(dev))
    _check(rc, "tbpm_propagate_qe")
    return corr, norm2, qe


def tbpm_haydock(H: Hamiltonian, sites, n_iter: int, workspace: Optional[torch.Tensor] = None):
    """NEXT-2: recursion coefficients (a [n_site][n_iter] = a_0.., b [n_site][n_iter] = b_1..) from the given host sites."""
    dev = H.device
    sites = torch.as_tensor(sites, dtype=torch.int64, device="cpu").contiguous()
    n_site = sites.numel()
    if workspace is None:
        workspace = _bytes(tbpm_propagate_bytes(H, n_site), dev)
    a = torch.zeros((n_site, n_iter), dtype=torch.float64, device=dev)
    b = torch.zeros((n_site, n_iter), dtype=torch.float64, device=dev)
    with torch.cuda.device(dev):
        rc = lib().tbpm_haydock(H.handle, C.c_void_p(sites.data_ptr()), n_site, n_iter, _ptr(a), _ptr(b), _ptr(workspace),
                                workspace.numel(), _stream(dev))
    _check(rc, "tbpm_haydock")
    return a, b


def tbpm_fermi_coeff(beta: float, mu: float, rescale: float, one_minus: bool = False, tol: float = 1e-13, kcap: int = 8192) -> torch.Tensor:
    """Host only: real Chebyshev coefficients [K] of the Fermi operator (or of 1 - f) on [-rescale, rescale]."""
    buf = torch.empty(kcap, dtype=torch.complex128)
    K = C.c_int(0)
    _check(lib().tbpm_fermi_coeff(beta, mu, rescale, int(one_minus), tol, kcap, C.byref(K), C.c_void_p(buf.data_ptr())), "tbpm_fermi_coeff")
    return buf[: K.value].real.clone()


def tbpm_corr_ac(H: Hamiltonian, Ja: Hamiltonian, Jb: Hamiltonian, psi0: torch.Tensor, n_step: int, dt: float, rescale: float, beta: float,
                 mu: float) -> torch.Tensor:
    """NEXT-4: corr complex128 [n_state][n_step + 1], entry n = <psi2(n dt)|J_a|psi1(n dt)>."""
    _need_cuda(psi0)
    dev = H.device
    psi0 = psi0.contiguous()
    n_state = psi0.shape[0]
    wb = C.c_size_t(0)
    _check(lib().tbpm_corr_ac_bytes(H.handle, n_state, C.byref(wb)), "tbpm_corr_ac_bytes")
    ws = _bytes(wb.value, dev)
    corr = torch.zeros((n_state, n_step + 1), dtype=torch.complex128, device=dev)
    with torch.cuda.device(dev):
        rc = lib().tbpm_corr_ac(H.handle, Ja.handle, Jb.handle, _ptr(psi0), n_state, n_step, dt, rescale, beta, mu, _ptr(corr), _ptr(ws),
                                ws.numel(), _stream(dev))
    _check(rc, "tbpm_corr_ac")
    return corr


def tbpm_corr_dp(H: Hamiltonian, rho_a: torch.Tensor, rho_b: torch.Tensor, psi0: torch.Tensor, n_step: int, dt: float, rescale: float,
                 beta: float, mu: float) -> torch.Tensor:
    """NEXT-4: corr complex128 [n_state][n_step + 1], entry n = <psi2(n dt)| rho_a * psi1(n dt)>; rho_a, rho_b complex128 [n_orb] on the device."""
    _need_cuda(psi0, rho_a, rho_b)
    dev = H.device
    # torch's conj() is lazy: resolve it, the library reads the raw (re, im) pairs
    psi0, rho_a, rho_b = psi0.resolve_conj().contiguous(), rho_a.resolve_conj().contiguous(), rho_b.resolve_conj().contiguous()
    assert rho_a.dtype == torch.complex128 and rho_a.numel() == H.n_orb and rho_b.numel() == H.n_orb
    n_state = psi0.shape[0]
    wb = C.c_size_t(0)
    _check(lib().tbpm_corr_ac_bytes(H.handle, n_state, C.byref(wb)), "tbpm_corr_ac_bytes")
    ws = _bytes(wb.value, dev)
    corr = torch.zeros((n_state, n_step + 1), dtype=torch.complex128, device=dev)
    with torch.cuda.device(dev):
        rc = lib().tbpm_corr_dp(H.handle, _ptr(rho_a), _ptr(rho_b), _ptr(psi0), n_state, n_step, dt, rescale, beta, mu, _ptr(corr), _ptr(ws),
                                ws.numel(), _stream(dev))
    _check(rc, "tbpm_corr_dp")
    return corr


def tbpm_haydock_ldos(a: torch.Tensor, b: torch.Tensor, energy: torch.Tensor, eta: float) -> torch.Tensor:
    """LDOS [n_site][n_energy] from the recursion coefficients (device tensors as returned by tbpm_haydock) by the continued fraction."""
    _need_cuda(a, b, energy)
    a, b, energy = a.contiguous(), b.contiguous(), energy.to(torch.float64).contiguous()
    n_site, n_iter = a.shape
    out = torch.zeros((n_site, energy.numel()), dtype=torch.float64, device=a.device)
    with torch.cuda.device(a.device):
        _check(lib().tbpm_haydock_ldos(_ptr(a), _ptr(b), n_site, n_iter, _ptr(energy), energy.numel(), eta, _ptr(out), _stream(a.device)),
               "tbpm_haydock_ldos")
    return out


def tbpm_dos(corr: torch.Tensor, dt: float, rescale: float):
    """corr complex128 [n_state][n_step] on the device -> (energy, dos), float64 [2 n_step + 1] each (tbpm.h: NEXT-1)."""
    _need_cuda(corr)
    corr = corr.contiguous()
    n_state, n_step = (1, corr.shape[0]) if corr.dim() == 1 else corr.shape
    energy = torch.zeros(2 * n_step + 1, dtype=torch.float64, device=corr.device)
    dos = torch.zeros_like(energy)
    with torch.cuda.device(corr.device):
        _check(lib().tbpm_dos(_ptr(corr), n_state, n_step, dt, rescale, _ptr(energy), _ptr(dos), _stream(corr.device)), "tbpm_dos")
    return energy, dos


def tbpm_get_state(H: Hamiltonian, workspace: torch.Tensor, state: int) -> torch.Tensor:
    out = torch.empty(max(H.n_orb, 1), dtype=torch.complex128, device=H.device)
    with torch.cuda.device(H.device):
        _check(lib().tbpm_get_state(H.handle, _ptr(workspace), state, _ptr(out), _stream(H.device)), "tbpm_get_state")
    return out[: H.n_orb]


def tbpm_last_launch_count(H: Hamiltonian) -> int:
    return int(lib().tbpm_last_launch_count(H.handle))


def tbpm_set_option(H: Hamiltonian, option: int, value: int) -> None:
    _check(lib().tbpm_set_option(H.handle, option, value), "tbpm_set_option")


def tbpm_total_launch_count() -> int:
    return int(lib().tbpm_total_launch_count())


def tbpm_corr_host_bytes(n_orb: int, n_hop: int, has_onsite: bool, n_state: int, n_step: int, flags: int = 0) -> int:
    b = C.c_size_t(0)
    _check(lib().tbpm_corr_host_bytes(n_orb, n_hop, int(has_onsite), n_state, n_step, flags, C.byref(b)), "tbpm_corr_host_bytes")
    return b.value


def tbpm_corr_host(n_orb: int, onsite, hop_i, hop_j, hop_val, psi0, n_step: int, dt: float, rescale: float, arena: torch.Tensor,
                   corr: torch.Tensor, norm2: Optional[torch.Tensor] = None, flags: int = 0):
    """End to end with HOST tensors (pinned for full copy bandwidth); `arena` is a device uint8 buffer of
    tbpm_corr_host_bytes().  Returns (h2d_bytes, d2h_bytes)."""
    for t in (hop_i, hop_j, hop_val, psi0, corr):
        assert not t.is_cuda and t.is_contiguous()
    _need_cuda(arena)
    up, down = C.c_size_t(0), C.c_size_t(0)
    dev = arena.device
    with torch.cuda.device(dev):
        rc = lib().tbpm_corr_host(n_orb, _ptr(onsite), hop_i.numel(), _ptr(hop_i), _ptr(hop_j), _ptr(hop_val), flags, _ptr(psi0),
                                  psi0.shape[0], n_step, dt, rescale, _ptr(corr), _ptr(norm2), _ptr(arena), arena.numel(),
                                  _stream(dev), C.byref(up), C.byref(down))
    _check(rc, "tbpm_corr_host")
    return up.value, down.value
