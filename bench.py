#!/usr/bin/env python
"""bench.py -- throughput of the TBPM hot path on B200 (one JSON line on stdout, rank 0).

A bench "step" is one pass of the whole hot path (every row) over one batch of synthetic input:
tbpm_build (hop list -> CSR + kernel layout) followed by tbpm_propagate of ALL the workload's states over a fixed block of
`n_step_per_bench_step` time steps (coefficients, state set-up, K-1 fused Chebyshev-term kernels per time step and state
tile, per-step correlation + norm).  Inputs are resident in HBM when the timed region starts.
`value` = n_state * n_block * (K-1) * nnz / step time, summed over ranks.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1..5|5ldos|3qe|4ac|5dp|5haydock] [--block B] [--impl reference]

Default workload: BASELINE.json:configs[4] (cubic 256^3 + Anderson disorder, 16,777,216 orbitals x 32 states): the largest
single-GPU configuration, one of the >= 16 M-orbital configs `north_star` sets its target on.  The full run length of a
config (1024-2048 time steps) would make one bench step minutes long; every time step launches the same kernels on
the same buffers, so a block of 8 time steps (~1 s on cfg5) is the unit that is timed, and `config` says so.  At N = 1
the line also carries `per_workload`: cfg3, cfg4 and cfg5's 64-site LDOS leg measured in the same process for >= 5 s each.
Multi-GPU: states are independent, so every rank propagates its own batch of seeded states on a replica of
H (paper_2509_26309_b200/replicas.py); no data-path collective; scaling is weak.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
`--workload 3qe` (cfg3 + quasi-eigenstates at 2 energies, NEXT-3), `--workload 4ac` / `5dp` (AC-conductivity and dynamic-polarisation
correlations on cfg4's / cfg5's lattice, NEXT-4) and `--workload 5haydock` (Haydock recursion from cfg5's 64
sites, NEXT-2) time the two NEXT rows that have kernels of their own (one GPU, one JSON line with `roofline`).
"""
from __future__ import annotations

import argparse
import csv
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Chebyshev terms*nnz/sec (complex128)"
UNIT = "nnz*terms/s"
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="5", help="1..5 = BASELINE.json:configs[i-1]; 5ldos = config 5's 64-site LDOS leg")
    ap.add_argument("--block", type=int, default=0, help="time steps per bench step (default: 8; 64 for cfg2, 256 for cfg1)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target wall time of the cpu_baseline sample")
    ap.add_argument("--per-workload-seconds", type=float, default=5.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-workload", action="store_true")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(workload_name: str, K: int):
    """Average DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per term launch over one time step, from the ncu
    captures of THIS round's final kernels (profiles/r2_terms.md: all 20 launches of a time step per workload) summarised in
    profiles/r2_dram_traffic.csv (one row per workload and kind of launch: first term, first flush, plain term, flush, last
    term).  None when the file has no row for the workload."""
    if not os.path.exists(TRAFFIC_CSV) or K < 4:
        return None, None
    rows = {}
    src = None
    with open(TRAFFIC_CSV) as f:
        for r in csv.DictReader(l for l in f if not l.startswith("#")):
            if r["workload"] == workload_name.split(":")[0] + ("-ldos" if workload_name.endswith("-ldos") else ""):
                rows[r["launch"]] = float(r["dram_mbytes"])
                src = r["source"]
    if "step_total" in rows:                                              # two terms per launch (cfg4): all launches of a time step of 20 terms
        return (1e6 * rows["step_total"] / (K - 1), src) if K == 21 else (None, None)
    need = ("first", "first_flush", "plain", "flush", "last")
    if any(k not in rows for k in need):
        return None, None
    n_flush = len([k for k in range(3, K - 1) if k % 3 == 2])
    n_plain = (K - 1) - 3 - n_flush
    avg = 1e6 * (rows["first"] + rows["first_flush"] + rows["last"] + n_flush * rows["flush"] + n_plain * rows["plain"]) / (K - 1)
    return avg, src


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                                          "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def default_block(cfg: int) -> int:
    return {1: 256, 2: 64}.get(cfg, 8)


def parse_tag(tag: str):
    return int(tag[0]), tag.lower().endswith("ldos")


# ---------------------------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on a bounded sample of the same workload
# ---------------------------------------------------------------------------------------------------------------------
def oracle_sample(w, ldos, seconds, steps=1, warmup=0, serial=False):
    """Times oracle.propagate (OpenMP row form, all host cores) on ONE state of the workload for m time steps chosen so
    that one sample takes about `seconds`.  Returns a dict (value nnz*terms/s, ms per sample, description, cores); with
    serial=True also the single-thread hop-list form (the authoritative statement of PAPER.md:437-443) over one time step."""
    import numpy as np
    import oracle
    hi, hj, hv = w.hop_i.cpu().numpy(), w.hop_j.cpu().numpy(), w.hop_val.cpu().numpy()
    on = None if w.onsite is None else w.onsite.cpu().numpy()
    if ldos:
        psi0 = np.zeros((1, w.n_orb), dtype=np.complex128)
        psi0[0, int(w.sites()[0])] = 1.0
    else:
        psi0 = w.psi0(device="cpu", n_state=1).numpy()
    K = len(oracle.cheb_coeff(w.rescale * w.dt))
    nnz = w.nnz

    def one(m, form="csr"):
        t0 = time.perf_counter()
        oracle.propagate(w.n_orb, on, hi, hj, hv, psi0, m, w.dt, w.rescale, form=form)
        return time.perf_counter() - t0

    t1 = one(1)
    t2 = one(2)
    per_step = max(t2 - t1, 1e-6)                           # the CSR build inside propagate is in both
    m = max(1, min(int((seconds - (t1 - per_step)) / per_step), 4096))
    times = []
    for it in range(warmup + steps):
        t = one(m)
        if it >= warmup:
            times.append(t)
    t = max(times)
    out = {"value": m * (K - 1) * nnz / t, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
           "sample": f"1 state x {m} time steps ({m * (K - 1)} H-applications) of the full-size lattice, oracle row form incl. its CSR build",
           "ms_per_sample": 1e3 * statistics.mean(times)}
    if serial:
        ts = one(1, form="hops")
        out["serial_hop_form"] = {"value": (K - 1) * nnz / ts, "unit": UNIT, "cores": 1,
                                  "sample": "1 state x 1 time step, single-thread hop-list form (oracle_propagate)"}
    return out


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2509_26309_b200 import workloads as W
    cfg, ldos = parse_tag(args.workload)
    w = W.make_workload(cfg, device="cpu")
    n_state = w.ldos_n_site if ldos else w.n_state
    r = oracle_sample(w, ldos, args.cpu_seconds, steps=max(1, args.steps), warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["ms_per_sample"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128", "data": "synthetic",
            "config": {"workload": w.name + ("-ldos" if ldos else ""), "n_orb": w.n_orb, "nnz": w.nnz, "n_state": n_state, "n_step": w.n_step,
                       "n_step_per_bench_step": args.block or default_block(cfg), "rescale": w.rescale, "tau": math.pi},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------------
class Runner:
    """One workload on one device: builds, propagates a block of time steps, reports rates and the roofline figures."""

    def __init__(self, tag, dev, shard, block):
        import torch
        from paper_2509_26309_b200 import tbpm, workloads as W
        self.torch, self.tbpm = torch, tbpm
        self.cfg, self.ldos = parse_tag(tag)
        self.dev = dev
        self.w = w = W.make_workload(self.cfg, device=dev)
        self.n_state = w.ldos_n_site if self.ldos else w.n_state
        self.block = block or default_block(self.cfg)
        # each rank propagates its own batch of seeded states (sub-streams shard.first_state ...); H is replicated
        self.psi0 = None if self.ldos else w.psi0(device=dev, n_state=self.n_state, first_state=shard.first_state)
        self.sites = W.ldos_sites(w.n_orb, self.n_state * shard.world)[shard.first_state: shard.first_state + self.n_state] if self.ldos else None
        self.K = len(tbpm.tbpm_cheb_coeff(w.rescale * w.dt))
        self.corr = torch.zeros((self.n_state, self.block), dtype=torch.complex128, device=dev)
        self.norm2 = torch.zeros((self.n_state, self.block), dtype=torch.float64, device=dev)
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)          # > L2 (126 MB)
        self.ws = None
        self.H = None
        self.name = w.name + ("-ldos" if self.ldos else "")

    def step(self, ev=None):
        torch, tbpm, w = self.torch, self.tbpm, self.w
        self.flush.fill_(1)                                                # evict L2 between iterations (untimed)
        if ev is not None:
            ev[0].record()
        H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val, 0)
        if self.ws is None:
            self.ws = torch.empty(tbpm.tbpm_propagate_bytes(H, self.n_state), dtype=torch.uint8, device=self.dev)
        if ev is not None:
            ev[1].record()
        if self.ldos:
            lc, ln, _ = tbpm.tbpm_ldos(H, self.sites, self.block, w.dt, w.rescale, workspace=self.ws)
            self.corr.copy_(lc); self.norm2.copy_(ln)
        else:
            tbpm.tbpm_propagate(H, self.psi0, self.block, w.dt, w.rescale, workspace=self.ws, corr=self.corr, norm2=self.norm2)
        if ev is not None:
            ev[2].record()
        self.H = H

    def units_per_step(self):
        return self.n_state * self.block * (self.K - 1) * self.H.nnz

    def roofline(self, prop_ms_per_step, peak, peak_src):
        """Algorithmic bytes (matrix as stored + 3 vectors) against the measured launch time of the fused term.
        The matrix bytes are those of the layout the running kernel reads: on the lattices the builder recognises (tiles of 8
        states; short rows with one real value for tiles of one state) that is a few bytes per row, not the general kernel layout; the figure with the general layout is given beside it."""
        H, w = self.H, self.w
        tile = min(8, 1 << max(self.n_state - 1, 0).bit_length())
        n_tile = -(-self.n_state // tile)
        term_launches = n_tile * self.block * (self.K - 1)
        avg_launch_s = prop_ms_per_step * 1e-3 / term_launches
        lattice = (tile == 8 and H.lattice_kind in (2, 3)) or (tile == 1 and H.lattice_kind == 4)
        m_launch = H.lattice_bytes_per_term if lattice else H.matrix_bytes_per_term     # what ONE launch reads of H
        bytes_tile = m_launch + 48 * w.n_orb * min(tile, self.n_state)                    # one launch = one tile of states
        bytes_term_strict = m_launch + 48 * w.n_orb * self.n_state                        # one term for ALL states, matrix counted once
        bytes_term_general = H.matrix_bytes_per_term + 48 * w.n_orb * self.n_state        # the same with the general kernel layout
        achieved_strict = bytes_term_strict / (avg_launch_s * n_tile) / 1e9
        achieved_tile = bytes_tile / avg_launch_s / 1e9
        traffic, tsrc = ncu_traffic(w.name + ("-ldos" if self.ldos else ""), self.K)
        kernel = {2: "k_term_l3 (fused Chebyshev term, three-dimensional lattice kernel, term_l3.cu)",
                  3: "k_pair_sq (TWO fused Chebyshev terms per launch, square lattice with in-line hoppings, term_sq2.cu)",
                  4: "k_term_n16 (fused Chebyshev term, short rows with 16-bit column offsets, term_n16.cu)"}.get(
                      H.lattice_kind if lattice else 0, "k_term_ph (fused Chebyshev term, term_ph.cuh)")
        return {"bound": "hbm", "kernel": kernel,
                "achieved": achieved_strict, "peak": peak, "unit": "GB/s", "frac": achieved_strict / peak,
                "traffic": traffic, "traffic_source": tsrc, "peak_source": peak_src,
                "frac_traffic": None if traffic is None else traffic / avg_launch_s / 1e9 / peak,
                "bytes_per_launch": bytes_tile, "avg_launch_us": avg_launch_s * 1e6, "launches_per_step": term_launches,
                "matrix_bytes_per_launch": m_launch, "matrix_bytes_general_layout": H.matrix_bytes_per_term,
                "count": "strict: matrix bytes the running kernel's layout stores + 3*16*N*n_state once per term for all states "
                         "(SURVEY 8(d)), over the time of the n_tile launches that make one term; *_per_tile counts the matrix once "
                         "per launch (one tile of <= 8 states); *_general_layout counts the general kernel layout (orp/ocol/oidx/diag), "
                         "which the lattice kernels do not read",
                "achieved_per_tile": achieved_tile, "frac_per_tile": achieved_tile / peak, "n_tile": n_tile,
                "frac_general_layout": bytes_term_general / (avg_launch_s * n_tile) / 1e9 / peak,
                "frac_of_nominal_8000": achieved_strict / 8000.0,
                "note": "avg launch = CUDA-event time of tbpm_propagate / TERMS x tiles (includes the <1% of tiny kernels; on cfg4 one "
                        "launch computes two terms, so this is the time per term, and a pair moves 4 vectors where the count has 6: "
                        "frac can exceed the traffic-based figure); traffic = "
                        "DRAM bytes per launch measured by ncu (read + write) averaged over the launches of a time step, "
                        "frac_traffic = traffic / avg launch / peak"}


def timed_steps(r, n, barrier):
    torch = r.torch
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n)]
    for i in range(n):
        r.step(evs[i])
    barrier()
    step_ms = [e[0].elapsed_time(e[2]) for e in evs]                      # device time, build + propagate
    prop_ms = [e[1].elapsed_time(e[2]) for e in evs]
    return sum(step_ms), sum(prop_ms)


def main_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_26309_b200 import tbpm, replicas

    rank, world, local = replicas.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the TBPM path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peak, peak_src = load_peaks()

    def barrier():
        replicas.barrier(dev)

    cfg, ldos = parse_tag(args.workload)
    probe_n_state = None

    def make(tag, block):
        from paper_2509_26309_b200 import workloads as W
        c, l = parse_tag(tag)
        n_state = W._FULL[c].get("ldos", 0) if l else W._FULL[c]["n_state"]
        return Runner(tag, dev, replicas.weak_shard(n_state, rank, world), block)

    r = make(args.workload, args.block)
    for _ in range(max(args.warmup, 0)):
        r.step()
    barrier()
    launches0 = tbpm.tbpm_total_launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    total_ms, prop_ms = timed_steps(r, args.steps, barrier)
    clocks = sampler.stop() if sampler else None
    launches = tbpm.tbpm_total_launch_count() - launches0
    total_ms, prop_ms = replicas.max_over_ranks([total_ms, prop_ms], dev)
    value = replicas.whole_job_rate(args.steps * r.units_per_step(), total_ms * 1e-3, dev)
    norm_dev = replicas.max_over_ranks([float((r.norm2 - 1).abs().max())], dev)[0]
    all_corr = replicas.gather_corr(r.corr, replicas.weak_shard(r.n_state, rank, world))
    gathered_ok = None
    if rank == 0:
        gathered_ok = bool(all_corr is not None and tuple(all_corr.shape) == (world * r.n_state, r.block) and
                           bool(torch.isfinite(torch.view_as_real(all_corr)).all()))
    w, H = r.w, r.H
    roofline = r.roofline(prop_ms / args.steps, peak, peak_src)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128", "data": "synthetic",
            "config": {"workload": r.name, "n_orb": w.n_orb, "nnz": H.nnz, "n_state": r.n_state, "n_step": w.n_step,
                       "n_step_per_bench_step": r.block, "K": r.K, "rescale": w.rescale, "tau": math.pi, "tile": 8, "n_table": H.n_table,
                       "matrix_bytes_per_term": H.matrix_bytes_per_term,
                       "l2": "256 MB flush between iterations; working set > L2", "ldos": ldos,
                       "parallelism": f"replicas x{world}: each rank its own {r.n_state} states (paper_2509_26309_b200/replicas.py)"},
            "ms_build": (total_ms - prop_ms) / args.steps, "ms_propagate": prop_ms / args.steps,
            "h_apps_per_s": value / H.nnz, "ms_per_time_step": prop_ms / args.steps / r.block,
            "max_norm_dev": norm_dev, "norm_ok": bool(norm_dev <= 1e-12), "gathered_corr_ok": gathered_ok,
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}

    # end to end through the C ABI with HOST buffers: H2D of the hop list and psi0, build, propagate, D2H of corr/norm2
    if not args.no_e2e and not ldos:
        hw = {k: getattr(w, k).cpu().pin_memory() for k in ("hop_i", "hop_j", "hop_val")}
        hon = None if w.onsite is None else w.onsite.cpu().pin_memory()
        hpsi = r.psi0.cpu().pin_memory()
        hcorr = torch.zeros((r.n_state, r.block), dtype=torch.complex128).pin_memory()
        hnorm = torch.zeros((r.n_state, r.block), dtype=torch.float64).pin_memory()
        dev_corr = r.corr.clone()
        r.ws = None                                                        # the arena below holds its own workspace
        torch.cuda.empty_cache()
        arena = torch.empty(tbpm.tbpm_corr_host_bytes(w.n_orb, w.n_hop, hon is not None, r.n_state, r.block, 0), dtype=torch.uint8, device=dev)
        up = down = 0
        e2e_t = []
        for i in range(1 + max(1, min(args.steps, 3))):
            barrier()
            t0 = time.perf_counter()
            up, down = tbpm.tbpm_corr_host(w.n_orb, hon, hw["hop_i"], hw["hop_j"], hw["hop_val"], hpsi, r.block, w.dt, w.rescale, arena,
                                           hcorr, hnorm, 0)
            if i > 0:
                e2e_t.append(time.perf_counter() - t0)
        te = replicas.max_over_ranks([sum(e2e_t)], dev)[0]
        line["e2e"] = {"value": replicas.sum_over_ranks([len(e2e_t) * r.units_per_step()], dev)[0] / te, "unit": UNIT,
                       "h2d_bytes_per_step": int(up), "d2h_bytes_per_step": int(down), "ms_per_step": 1e3 * te / len(e2e_t),
                       "max_abs_diff_vs_device_path": float((hcorr.to(dev) - dev_corr).abs().max()),
                       "api": "tbpm_corr_host: pinned host hop list + psi0 -> H2D, build, propagate, D2H of corr/norm2"}
        del arena, hpsi, hw

    # the other >= 16 M-orbital workloads, in the same process, for >= per_workload_seconds each (sustained clocks)
    if world == 1 and not args.no_per_workload and args.workload == "5":
        per = [{"workload": r.name, "value": value, "frac": roofline["frac"], "frac_per_tile": roofline["frac_per_tile"],
                "frac_general_layout": roofline["frac_general_layout"], "frac_traffic": roofline["frac_traffic"], "kernel": roofline["kernel"],
                "avg_launch_us": roofline["avg_launch_us"], "clocks": clocks, "max_norm_dev": norm_dev,
                "seconds": total_ms * 1e-3, "n_step_per_bench_step": r.block}]
        del r
        torch.cuda.empty_cache()
        for tag in ("3", "4", "5ldos"):
            q = make(tag, args.block)
            for _ in range(3):
                q.step()
            barrier()
            smp = ClockSampler(local)
            tot = prp = 0.0
            n = 0
            while tot * 1e-3 < args.per_workload_seconds:
                a, b = timed_steps(q, 2, barrier)
                tot += a; prp += b; n += 2
            ck = smp.stop()
            rf = q.roofline(prp / n, peak, peak_src)
            nd = float((q.norm2 - 1).abs().max())
            per.append({"workload": q.name, "value": n * q.units_per_step() / (tot * 1e-3), "frac": rf["frac"], "frac_per_tile": rf["frac_per_tile"],
                        "frac_general_layout": rf["frac_general_layout"], "frac_traffic": rf["frac_traffic"],
                        "avg_launch_us": rf["avg_launch_us"], "bytes_per_launch": rf["bytes_per_launch"], "kernel": rf["kernel"],
                        "traffic": rf["traffic"], "clocks": ck, "max_norm_dev": nd, "norm_ok": bool(nd <= 1e-12),
                        "seconds": tot * 1e-3, "n_step_per_bench_step": q.block})
            del q
            torch.cuda.empty_cache()
        line["per_workload"] = per

    if rank == 0 and not args.no_cpu_baseline:
        from paper_2509_26309_b200 import workloads as W
        wc = W.make_workload(cfg, device="cpu")
        line["cpu_baseline"] = oracle_sample(wc, ldos, args.cpu_seconds, serial=True)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------------------------------
# the NEXT rows: quasi-eigenstates (3qe), AC-conductivity correlation (4ac) and the Haydock recursion (5haydock); one GPU
# ---------------------------------------------------------------------------------------------------------------------
def main_next(args):
    import torch
    from paper_2509_26309_b200 import tbpm, workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the TBPM path has no CPU fallback")
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, peak_src = load_peaks()
    cfg = int(args.workload[0])
    haydock = args.workload.endswith("haydock")
    ac = args.workload.endswith("ac")
    dp = args.workload.endswith("dp")
    w = W.make_workload(cfg, device=dev)
    H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val, 0)
    block = args.block or 8
    K = len(tbpm.tbpm_cheb_coeff(w.rescale * w.dt))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    if ac:
        # NEXT-4: AC-conductivity correlation <psi2(t)|J_x|psi1(t)> on the lattice of cfg4 (Fermi-operator Chebyshev filters, two states
        # propagated side by side, one current-operator product per time step); beta = 2 / |t|, mu = 0.5 |t|
        n_state, beta, mu = w.n_state, 2.0, 0.5
        psi0 = w.psi0(device=dev, n_state=n_state)
        _, ji, jj, jv = W.square_current_hops(w.meta["Lx"], w.meta["Ly"], 0, phi_den=w.meta["phi_den"], device=dev)
        J = tbpm.tbpm_build(w.n_orb, None, ji, jj, jv)
        run = lambda: tbpm.tbpm_corr_ac(H, J, J, psi0, block, w.dt, w.rescale, beta, mu)
        Kf = len(tbpm.tbpm_fermi_coeff(beta, mu, w.rescale, False)); Kg = len(tbpm.tbpm_fermi_coeff(beta, mu, w.rescale, True))
        apps = (Kf - 1) + (Kg - 1) + 2 * block * (K - 1)             # H applications per state
        units = n_state * apps * H.nnz
        mat = H.lattice_bytes_per_term if H.lattice_kind in (2, 3) else H.matrix_bytes_per_term
        vec = 16 * w.n_orb * n_state
        bytes_step = apps * (mat + 3 * vec) + (J.matrix_bytes_per_term + 2 * vec) + (block + 1) * (J.matrix_bytes_per_term + 3 * vec)
        what = (f"AC-conductivity correlation: Fermi filters of {Kf} and {Kg} Chebyshev terms, then {block} time steps of two states "
                "(k_pair_sq: two Chebyshev terms per launch, as in the filters) with one current-operator product fused with the dot product per step")
        count = ("per H application: matrix bytes of the running kernel's layout + 3 vectors; J_b psi0: current matrix + 2 vectors; per "
                 "<psi2|J_a|psi1>: current matrix + 3 vectors (workspace allocation included in the time)")
    elif dp:
        # NEXT-4, second half: dynamic-polarisation correlation <psi2(t)|rho(q)|psi1(t)> on the lattice of cfg5, one tile of 8 states,
        # q = (2 pi / L)(1, 0, 2); the density operators are diagonal, so there is no second matrix
        import math
        n_state, beta, mu, L = 8, 0.5, 1.0, w.meta["L"]
        psi0 = w.psi0(device=dev, n_state=n_state)
        idx = torch.arange(w.n_orb, device=dev)
        ph = (2 * math.pi / L) * (1.0 * (idx % L) + 2.0 * (idx // (L * L))).to(torch.float64)
        rho = torch.complex(torch.cos(ph), torch.sin(ph))
        rho_c = rho.conj().resolve_conj().contiguous()
        run = lambda: tbpm.tbpm_corr_dp(H, rho, rho_c, psi0, block, w.dt, w.rescale, beta, mu)
        Kf = len(tbpm.tbpm_fermi_coeff(beta, mu, w.rescale, False)); Kg = len(tbpm.tbpm_fermi_coeff(beta, mu, w.rescale, True))
        apps = (Kf - 1) + (Kg - 1) + 2 * block * (K - 1)
        units = n_state * apps * H.nnz
        mat = H.lattice_bytes_per_term if H.lattice_kind in (2, 3) else H.matrix_bytes_per_term
        vec = 16 * w.n_orb * n_state
        bytes_step = apps * (mat + 3 * vec) + (16 * w.n_orb + 2 * vec) + (block + 1) * (16 * w.n_orb + 2 * vec)
        what = (f"dynamic-polarisation correlation: Fermi filters of {Kf} and {Kg} Chebyshev terms, then {block} time steps of two states "
                "(k_term_l3) with one diagonal density-operator product fused with the dot product per step (k_diag_dot)")
        count = ("per H application: matrix bytes of the running kernel's layout + 3 vectors; rho_b psi0: diagonal + 2 vectors; per "
                 "<psi2|rho_a|psi1>: diagonal + 2 vectors (workspace allocation included in the time)")
    elif haydock:
        n_state = w.ldos_n_site
        sites = W.ldos_sites(w.n_orb, n_state)
        ws = torch.empty(tbpm.tbpm_propagate_bytes(H, n_state), dtype=torch.uint8, device=dev)
        run = lambda: tbpm.tbpm_haydock(H, sites, block, workspace=ws)
        units = n_state * block * H.nnz                              # H applications x nnz
        tile = 8
        mat = H.lattice_bytes_per_term if H.lattice_kind in (2, 3) else H.matrix_bytes_per_term
        # per recursion level and tile: H u (matrix, gather u, write t) + update (read t, u, u_prev, write u_next): matrix + 6 vectors
        bytes_step = (n_state // tile) * block * (mat + 6 * 16 * w.n_orb * tile)
        what = "Haydock recursion: H u fused with <u|H u> (k_term_l3, last-term shape) + three-vector update fused with the norm (k_haydock_update)"
        count = "per level and tile of 8 sites: matrix bytes of the running kernel's layout + 6 vectors (gather u, write t; read t, u, u_prev, write u_next)"
    else:
        n_state = w.n_state
        psi0 = w.psi0(device=dev, n_state=n_state)
        energies = [0.0, 0.5 * w.rescale]
        run = lambda: tbpm.tbpm_propagate_qe(H, psi0, energies, block, w.dt, w.rescale)
        units = n_state * block * (K - 1) * H.nnz
        # per time step: the K - 1 terms (matrix + 3 vectors each) + the accumulation sweep (read psi', read + write n_E vectors)
        mat = H.lattice_bytes_per_term if (H.lattice_kind == 4 and n_state == 1) else H.matrix_bytes_per_term
        bytes_step = block * ((K - 1) * (mat + 48 * w.n_orb * n_state) + (1 + 2 * len(energies)) * 16 * w.n_orb * n_state)
        what = "propagation + quasi-eigenstates at 2 energies: k_term_n16 / k_term_ph per term, k_qe_axpy once per time step"
        count = "per time step: (K - 1) x (matrix + 3 vectors) + (1 + 2 n_E) vectors of the accumulation sweep (workspace allocation and export included in the time)"
    for _ in range(max(args.warmup, 1)):
        run()
    torch.cuda.synchronize()
    launches0 = tbpm.tbpm_total_launch_count()
    sampler = ClockSampler(0)
    evs = []
    for _ in range(args.steps):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); out = run(); e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = sum(a.elapsed_time(b) for a, b in evs)
    achieved = args.steps * bytes_step / (ms * 1e-3) / 1e9
    line = {"metric": "Hamiltonian applications*nnz/sec (complex128)" if (haydock or ac or dp) else METRIC, "value": args.steps * units / (ms * 1e-3), "unit": UNIT,
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "complex128", "data": "synthetic",
            "config": {"workload": w.name + ("-ac" if ac else "-dp" if dp else "-haydock" if haydock else "-qe"), "n_orb": w.n_orb, "nnz": H.nnz, "n_state": n_state,
                       "n_step_per_bench_step": block, "what": what, "l2": "256 MB flush between iterations; working set > L2"},
            "gpu_launches": int(tbpm.tbpm_total_launch_count() - launches0), "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                         "peak_source": peak_src, "count": count}}
    if ac or dp:
        line["finite"] = bool(torch.isfinite(out.real).all() and torch.isfinite(out.imag).all())
    elif haydock:
        a, b = out
        line["finite"] = bool(torch.isfinite(a).all() and torch.isfinite(b).all() and (b > 0).all())
    else:
        line["max_norm_dev"] = float((out[1] - 1).abs().max())
    print(json.dumps(line))
    return 0


if __name__ == "__main__":
    a = parse_args()
    if a.workload.endswith("qe") or a.workload.endswith("haydock") or a.workload.endswith("ac") or a.workload.endswith("dp"):
        sys.exit(main_next(a))
    sys.exit(main_reference(a) if a.impl == "reference" else main_ours(a))
