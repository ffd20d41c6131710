"""Seeded synthetic input generators for the TBPM hot path (serves BOTH the CUDA library and the oracle).

This module holds none of the method's arithmetic: it only produces the *inputs* of the path --
hopping lists (each conjugate pair once, "hopping terms reduced by the conjugate relation
H_ij(R) = H_ji*(-R)"), optional real on-site energies (an orbital attribute), random-phase
initial states and LDOS site lists -- for the five lattices of BASELINE.json:configs.  It imports neither
`oracle/` nor the CUDA binding.  Everything is generated with torch ops on the device asked for
(torch is plumbing: memory + elementwise integer/float ops); random numbers come from a counter-based
64-bit hash of (seed, stream, sub-stream, index), so any element can be regenerated anywhere.

Readings of the paper fixed here (listed again in DESIGN.md):
  #12 random state      psi0_i = exp(i*theta_i)/sqrt(N), theta_i = 2*pi*u_i
  #20 honeycomb index   idx = (ia*Nb + ib)*2 + o ; hops A(ia,ib)-B(ia,ib), B(ia,ib)-A(ia+1,ib), B(ia,ib)-A(ia,ib+1)
                        (add_hopping((0,0,0),0,1,t), ((1,0,0),1,0,t), ((0,1,0),1,0,t))
  #21 vacancies         each site removed independently with prob p; survivors renumbered by stable compaction;
                        isolated survivors kept
  #22 Anderson          onsite_i = W*(u_i - 1/2)
  #23 Peierls           idx = y*Lx + x ; Landau gauge A=(0,Bx): <r'|H|r> = t*exp(+i*2*pi*phi*(x+x')/2*(y'-y)), x' unwrapped
  #24 cubic index       idx = (z*L + y)*L + x ; hops to +x,+y,+z
  #25 LDOS sites        n_site distinct sites from the seeded stream
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import torch

MASTER_SEED = 20250926
STREAM_PSI0, STREAM_DISORDER, STREAM_VACANCY, STREAM_LDOS = 1, 2, 3, 4

_M64 = (1 << 64) - 1


def _s64(v: int) -> int:
    """Python int (mod 2^64) -> the signed value torch.int64 holds for the same bit pattern."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


_GAMMA = _s64(0x9E3779B97F4A7C15)
_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right of int64 bit patterns."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def _mix64_t(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 tensors (wrapping multiply)."""
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def _mix64_i(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int, sub: int = 0) -> int:
    """64-bit key of one random stream (host integer arithmetic)."""
    k = _mix64_i(seed)
    k = _mix64_i(k ^ ((stream * 0x9E3779B97F4A7C15) & _M64))
    k = _mix64_i(k ^ ((sub * 0xD1B54A32D192ED03 + 0x2545F4914F6CDD1D) & _M64))
    return k


def counter_bits(key: int, start: int, n: int, device="cpu") -> torch.Tensor:
    """int64 tensor of n hashed 64-bit words for counters start..start+n-1 of stream `key`."""
    i = torch.arange(start + 1, start + n + 1, dtype=torch.int64, device=device)
    return _mix64_t(i * _GAMMA + _s64(key))


def counter_uniform(key: int, start: int, n: int, device="cpu") -> torch.Tensor:
    """float64 uniforms on [0,1) with 53 random bits."""
    b = _lsr(counter_bits(key, start, n, device), 11)
    return b.to(torch.float64) * (1.0 / 9007199254740992.0)


def random_phase_state(n_orb: int, state: int, seed: int = MASTER_SEED, device="cpu") -> torch.Tensor:
    """One state psi0_i = exp(i theta_i)/sqrt(N) (reading #12, BASELINE.json:configs[0]) -> complex128 [n_orb]."""
    u = counter_uniform(stream_key(seed, STREAM_PSI0, state), 0, n_orb, device)
    th = u * (2.0 * math.pi)
    a = 1.0 / math.sqrt(n_orb)
    return torch.complex(torch.cos(th) * a, torch.sin(th) * a)


def random_phase_states(n_orb: int, n_state: int, seed: int = MASTER_SEED, device="cpu", first_state: int = 0) -> torch.Tensor:
    out = torch.empty((n_state, n_orb), dtype=torch.complex128, device=device)
    for b in range(n_state):
        out[b] = random_phase_state(n_orb, first_state + b, seed, device)
    return out


def anderson_onsite(n_orb: int, W: float, seed: int = MASTER_SEED, device="cpu") -> torch.Tensor:
    """onsite_i = W*(u_i - 1/2) (reading #22)."""
    u = counter_uniform(stream_key(seed, STREAM_DISORDER), 0, n_orb, device)
    return (u - 0.5) * W


def ldos_sites(n_orb: int, n_site: int, seed: int = MASTER_SEED) -> torch.Tensor:
    """n_site distinct sites drawn from the seeded stream, redraw on repeat (reading #25) -> int64 [n_site] (host)."""
    key = stream_key(seed, STREAM_LDOS)
    sites, seen, c = [], set(), 0
    while len(sites) < n_site:
        u = float(counter_uniform(key, c, 1)[0])
        c += 1
        s = min(int(u * n_orb), n_orb - 1)
        if s not in seen:
            seen.add(s)
            sites.append(s)
    return torch.tensor(sites, dtype=torch.int64)


# ----------------------------------------------------------------------------------------------------------
# lattices: each returns (n_orb, hop_i int32[n_hop], hop_j int32[n_hop], hop_val complex128[n_hop]);
# entry (i, j, v) means <i|H|j> = v and the conjugate partner is implied (reading #13/#14).
# ----------------------------------------------------------------------------------------------------------

def honeycomb_hops(Na: int, Nb: int, t: float = -2.7, device="cpu"):
    """Graphene NN model of PAPER.md:738-765 on an Na x Nb periodic supercell (pbc (True, True, False))."""
    if Na < 3 or Nb < 3:
        raise ValueError("periodic extents must be >= 3 (wrap-around duplicates, reading #15)")
    ia = torch.arange(Na, dtype=torch.int64, device=device).view(Na, 1)
    ib = torch.arange(Nb, dtype=torch.int64, device=device).view(1, Nb)
    A = ((ia * Nb + ib) * 2).reshape(-1)            # orbital 0 of cell (ia, ib)
    B = A + 1
    A_a = ((((ia + 1) % Na) * Nb + ib) * 2).reshape(-1)   # A of cell (ia+1, ib)
    A_b = ((ia * Nb + ((ib + 1) % Nb)) * 2).reshape(-1)   # A of cell (ia, ib+1)
    # (0,0,0): 0->1 ; (1,0,0): 1->0 ; (0,1,0): 1->0   ( <i,0|H|j,R> )
    hop_i = torch.cat([A, B, B]).to(torch.int32)
    hop_j = torch.cat([B, A_a, A_b]).to(torch.int32)
    hop_val = torch.full((hop_i.numel(),), complex(t, 0.0), dtype=torch.complex128, device=device)
    return 2 * Na * Nb, hop_i, hop_j, hop_val


def apply_vacancies(n_orb: int, hop_i, hop_j, hop_val, p_remove: float, seed: int = MASTER_SEED):
    """Remove each site independently with probability p_remove; stable compaction; drop hops touching a removed
    site; keep isolated survivors (reading #21).  Returns (n_orb', hop_i', hop_j', hop_val', keep_mask)."""
    device = hop_i.device
    u = counter_uniform(stream_key(seed, STREAM_VACANCY), 0, n_orb, device)
    keep = u >= p_remove
    new_idx = torch.cumsum(keep.to(torch.int64), 0) - 1
    n_new = int(new_idx[-1].item()) + 1 if n_orb > 0 else 0
    hi, hj = hop_i.to(torch.int64), hop_j.to(torch.int64)
    ok = keep[hi] & keep[hj]
    hi2 = new_idx[hi[ok]].to(torch.int32)
    hj2 = new_idx[hj[ok]].to(torch.int32)
    return n_new, hi2, hj2, hop_val[ok].clone(), keep


def square_peierls_hops(Lx: int, Ly: int, t: float = -1.0, t2: float = 0.2, phi_num: int = 1, phi_den: int = 1024,
                        device="cpu"):
    """Square lattice, NN t and NNN t2, uniform flux phi = phi_num/phi_den flux quanta per plaquette, Landau gauge
    A = (0, Bx) (reading #23).  For a hop r -> r' the entry is <r'|H|r> = t_rr' * exp(+i 2 pi phi (x+x')/2 (y'-y)),
    x' = x + dx unwrapped.  Periodic-compatible iff phi*Lx is an integer."""
    if Lx < 3 or Ly < 3:
        raise ValueError("periodic extents must be >= 3")
    if (phi_num * Lx) % phi_den != 0:
        raise ValueError("phi*Lx must be an integer for periodic boundary conditions")
    y = torch.arange(Ly, dtype=torch.int64, device=device).view(Ly, 1)
    x = torch.arange(Lx, dtype=torch.int64, device=device).view(1, Lx)
    src = (y * Lx + x).reshape(-1)
    xf = x.to(torch.float64).expand(Ly, Lx).reshape(-1)
    phi = phi_num / phi_den

    def dest(dx, dy):
        return (((y + dy) % Ly) * Lx + ((x + dx) % Lx)).reshape(-1)

    def phase(dx, dy, amp):
        # (x + x')/2 * (y' - y) with x' = x + dx
        ang = (2.0 * math.pi * phi) * (xf + 0.5 * dx) * dy
        return torch.complex(torch.cos(ang) * amp, torch.sin(ang) * amp)

    his, hjs, hvs = [], [], []
    for dx, dy, amp in ((1, 0, t), (0, 1, t), (1, 1, t2), (-1, 1, t2)):
        his.append(dest(dx, dy))      # row  = r'
        hjs.append(src)               # col  = r
        hvs.append(phase(dx, dy, amp))
    hop_i = torch.cat(his).to(torch.int32)
    hop_j = torch.cat(hjs).to(torch.int32)
    hop_val = torch.cat(hvs)
    return Lx * Ly, hop_i, hop_j, hop_val


def square_current_hops(Lx: int, Ly: int, axis: int, t: float = -1.0, t2: float = 0.2, phi_num: int = 1, phi_den: int = 1024, device="cpu"):
    """Hop list of the current operator J_axis = i [H, r_axis] of square_peierls_hops' lattice (hbar = e = 1; NEXT-4): the entry
    <r'|J|r> = i * <r'|H|r> * (r' - r)_axis with the UNWRAPPED displacement of the hop; hops without a component along the axis are
    left out.  Hermitian like H, so the list holds each conjugate pair once and goes through tbpm_build / the oracle as it is."""
    n, hi, hj, hv = square_peierls_hops(Lx, Ly, t, t2, phi_num, phi_den, device)
    per = Lx * Ly
    disp = []
    for dx, dy in ((1, 0), (0, 1), (1, 1), (-1, 1)):               # the four hop families, in square_peierls_hops' order
        disp.append(torch.full((per,), float((dx, dy)[axis]), dtype=torch.float64, device=device))
    d = torch.cat(disp)
    keep = d != 0
    val = torch.complex(-hv.imag * d, hv.real * d)                 # i * v * d
    return n, hi[keep].contiguous(), hj[keep].contiguous(), val[keep].contiguous()


def cubic_hops(L: int, t: float = -1.0, device="cpu"):
    """Simple-cubic L^3 periodic, idx = (z*L + y)*L + x, hops to +x, +y, +z (reading #24)."""
    if L < 3:
        raise ValueError("periodic extents must be >= 3")
    z = torch.arange(L, dtype=torch.int64, device=device).view(L, 1, 1)
    y = torch.arange(L, dtype=torch.int64, device=device).view(1, L, 1)
    x = torch.arange(L, dtype=torch.int64, device=device).view(1, 1, L)
    src = ((z * L + y) * L + x).reshape(-1)
    dx = ((z * L + y) * L + (x + 1) % L).reshape(-1)
    dy = ((z * L + (y + 1) % L) * L + x).reshape(-1)
    dz = ((((z + 1) % L) * L + y) * L + x).reshape(-1)
    hop_i = torch.cat([src, src, src]).to(torch.int32)
    hop_j = torch.cat([dx, dy, dz]).to(torch.int32)
    hop_val = torch.full((hop_i.numel(),), complex(t, 0.0), dtype=torch.complex128, device=device)
    return L ** 3, hop_i, hop_j, hop_val


def square_range_hops(Lx: int, Ly: int, radius: float, n_phase: int = 1, device="cpu"):
    """Square lattice with a hop to EVERY site within `radius` (third-neighbour-style models with long rows: 12 neighbours
    at radius 2, 28 at 3, 48 at 4, 80 at 5).  Not one of BASELINE.json's configs: it exists to drive the kernels through rows
    longer than the 8 entries the configs have.  <r'|H|r> = 0.3/d^2 * exp(i(0.4 dx - 0.7 dy)) * exp(i 2 pi (x mod n_phase)/n_phase dy):
    n_phase sets the number of distinct values (table size).  Returns (n_orb, hop_i, hop_j, hop_val, row_sum) with
    row_sum = sum_j |H_ij| (the same for every row: a valid `rescale`)."""
    r = int(math.floor(radius))
    if Lx < 2 * r + 1 or Ly < 2 * r + 1:
        raise ValueError("periodic extents must exceed 2*radius (wrap-around duplicates, reading #15)")
    if Lx % n_phase != 0:
        raise ValueError("n_phase must divide Lx")
    y = torch.arange(Ly, dtype=torch.int64, device=device).view(Ly, 1)
    x = torch.arange(Lx, dtype=torch.int64, device=device).view(1, Lx)
    src = (y * Lx + x).reshape(-1)
    xf = (x % n_phase).to(torch.float64).expand(Ly, Lx).reshape(-1) * (2.0 * math.pi / n_phase)
    his, hjs, hvs = [], [], []
    row_sum = 0.0
    for dx in range(0, r + 1):
        for dy in range(-r, r + 1):
            if dx * dx + dy * dy > radius * radius or (dx == 0 and dy <= 0):
                continue                                     # each pair once: dx > 0, or dx == 0 and dy > 0
            amp = 0.3 / (dx * dx + dy * dy)
            ang = xf * dy + (0.4 * dx - 0.7 * dy)
            his.append((((y + dy) % Ly) * Lx + ((x + dx) % Lx)).reshape(-1))
            hjs.append(src)
            hvs.append(torch.complex(torch.cos(ang) * amp, torch.sin(ang) * amp))
            row_sum += 2.0 * amp
    return Lx * Ly, torch.cat(his).to(torch.int32), torch.cat(hjs).to(torch.int32), torch.cat(hvs), row_sum


def chain_hops(L: int, t: float = -1.0, device="cpu"):
    """1-D periodic chain (used for the closed-form DOS pin 1/(pi sqrt(4t^2-E^2)))."""
    if L < 3:
        raise ValueError("periodic extents must be >= 3")
    i = torch.arange(L, dtype=torch.int64, device=device)
    return L, i.to(torch.int32), ((i + 1) % L).to(torch.int32), torch.full((L,), complex(t, 0.0), dtype=torch.complex128, device=device)


# ----------------------------------------------------------------------------------------------------------
# the five workloads of BASELINE.json:configs (1-based ids as in SURVEY.md section 8(d))
# ----------------------------------------------------------------------------------------------------------

@dataclass
class Workload:
    name: str
    n_orb: int
    hop_i: torch.Tensor
    hop_j: torch.Tensor
    hop_val: torch.Tensor
    onsite: Optional[torch.Tensor]
    n_state: int
    n_step: int
    rescale: float
    seed: int = MASTER_SEED
    ldos_n_site: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def dt(self) -> float:
        """tau = rescale*dt = pi for every config (BASELINE.json:configs; reading #6)."""
        return math.pi / self.rescale

    @property
    def n_hop(self) -> int:
        return int(self.hop_i.numel())

    @property
    def nnz(self) -> int:
        return 2 * self.n_hop + (self.n_orb if self.onsite is not None else 0)

    def psi0(self, device=None, n_state=None, first_state=0) -> torch.Tensor:
        device = self.hop_i.device if device is None else device
        return random_phase_states(self.n_orb, self.n_state if n_state is None else n_state, self.seed, device, first_state)

    def sites(self) -> torch.Tensor:
        return ldos_sites(self.n_orb, self.ldos_n_site, self.seed)


_FULL = {
    1: dict(kind="honeycomb", Na=64, Nb=64, n_state=1, n_step=256, rescale=9.0),
    2: dict(kind="honeycomb", Na=1024, Nb=1024, W=1.0, n_state=4, n_step=1024, rescale=9.5),
    3: dict(kind="honeycomb", Na=4096, Nb=4096, vac=0.10, n_state=1, n_step=1024, rescale=9.0),
    4: dict(kind="square", Lx=4096, Ly=4096, phi_den=1024, n_state=8, n_step=2048, rescale=4.8),
    5: dict(kind="cubic", L=256, W=16.5, n_state=32, n_step=1024, rescale=15.0, ldos=64),
}


def make_workload(cfg: int, device="cpu", seed: int = MASTER_SEED, **override) -> Workload:
    """Workload `cfg` (1..5) of BASELINE.json:configs[cfg-1].  `override` may shrink the lattice (Na, Nb, Lx, Ly, L,
    phi_den, n_state, n_step) for tests; the structure (degree distribution, value distribution) is unchanged."""
    p = dict(_FULL[cfg])
    p.update(override)
    kind = p["kind"]
    onsite = None
    if kind == "honeycomb":
        n, hi, hj, hv = honeycomb_hops(p["Na"], p["Nb"], -2.7, device)
        name = f"cfg{cfg}:honeycomb{p['Na']}x{p['Nb']}"
        if p.get("vac"):
            n, hi, hj, hv, _ = apply_vacancies(n, hi, hj, hv, p["vac"], seed)
            name += f"-vac{p['vac']}"
        if p.get("W"):
            onsite = anderson_onsite(n, p["W"], seed, device)
            name += f"-W{p['W']}"
    elif kind == "square":
        n, hi, hj, hv = square_peierls_hops(p["Lx"], p["Ly"], -1.0, 0.2, 1, p["phi_den"], device)
        name = f"cfg{cfg}:square{p['Lx']}x{p['Ly']}-flux1/{p['phi_den']}"
    elif kind == "cubic":
        n, hi, hj, hv = cubic_hops(p["L"], -1.0, device)
        onsite = anderson_onsite(n, p["W"], seed, device) if p.get("W") else None
        name = f"cfg{cfg}:cubic{p['L']}^3-W{p.get('W', 0)}"
    else:
        raise ValueError(kind)
    return Workload(name=name, n_orb=n, hop_i=hi, hop_j=hj, hop_val=hv, onsite=onsite, n_state=p["n_state"],
                    n_step=p["n_step"], rescale=p["rescale"], seed=seed, ldos_n_site=p.get("ldos", 0), meta=p)
