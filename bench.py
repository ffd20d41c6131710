#!/usr/bin/env python
"""bench.py -- throughput of the TBPM hot path on B200 (one JSON line on stdout, rank 0).

A "step" is one pass of the whole hot path over one batch of synthetic input: tbpm_build (hop list -> CSR + kernel
layout) followed by tbpm_propagate over the workload's full n_step time steps for all its states (coefficients,
state set-up, K-1 fused Chebyshev-term kernels per time step, per-step correlation + norm).  Inputs are resident in
HBM when the timed region starts.  `value` = n_state * n_step * (K-1) * nnz / step time, summed over ranks.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1..5|5ldos] [--impl reference]

Default workload: BASELINE.json:configs[1] (honeycomb 1024x1024 + Anderson disorder, 4 states, 1024 steps).
Multi-GPU: states are independent, so every rank propagates its own batch of seeded states on a
replica of H; no data-path collective; scaling is weak.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
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


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="2", help="1..5 = BASELINE.json:configs[i-1]; 5ldos = config 5's 64-site LDOS leg")
    ap.add_argument("--n-step", type=int, default=0, help="override the workload's number of time steps (development only; "
                                                            "the JSON line then says so in config.n_step_override)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target wall time of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the fused term, MB, from the one `ncu --set full` capture per
# workload summarised in profiles/r1b_ncu_full_cfg2-5.md: (first term k=1, first flush k=2, plain term, flush, last term).
NCU_TRAFFIC_SRC = "profiles/r1b_ncu_full_cfg2-5.md (ncu --set full, one capture per workload; average over the launches of a time step)"
NCU_TRAFFIC_MB = {"cfg2": (279.2, 531.7, 414.6, 668.7, 694.5), "cfg3": (1384.0, 2330.0, 1868.0, 2815.0, 2839.0),
                  "cfg4": (5137.0, 9412.0, 7284.0, 11560.0, 11584.0), "cfg5": (5002.0, 9322.0, 7152.0, 11646.0, 12547.0)}


def ncu_traffic(workload_name: str, K: int):
    """Average DRAM bytes per term launch over one time step (K-1 launches: flush every third term), or None."""
    t = NCU_TRAFFIC_MB.get(workload_name.split(":")[0])
    if t is None or K < 4:
        return None
    first, first_flush, plain, flush, last = t
    n_flush = len([k for k in range(3, K - 1) if k % 3 == 2])
    n_plain = (K - 1) - 3 - n_flush
    return 1e6 * (first + first_flush + last + n_flush * flush + n_plain * plain) / (K - 1)


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


def workload_of(tag: str, device, rank: int, n_step_override: int):
    from paper_2509_26309_b200 import workloads as W
    ldos = tag.lower().endswith("ldos")
    cfg = int(tag[0])
    w = W.make_workload(cfg, device=device)
    n_step = n_step_override or w.n_step
    n_state = w.ldos_n_site if ldos else w.n_state
    return w, cfg, ldos, n_state, n_step


# ---------------------------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on a bounded sample of the same workload
# ---------------------------------------------------------------------------------------------------------------------
def oracle_sample(w, cfg_tag, seconds, steps=1, warmup=0):
    """Times oracle.propagate (OpenMP row form, all host cores) on ONE state of the workload for m time steps chosen so
    that one sample takes about `seconds`.  Returns (value nnz*terms/s, ms per sample, description, cores)."""
    import numpy as np
    import oracle
    hi, hj, hv = w.hop_i.cpu().numpy(), w.hop_j.cpu().numpy(), w.hop_val.cpu().numpy()
    on = None if w.onsite is None else w.onsite.cpu().numpy()
    if cfg_tag.endswith("ldos"):
        psi0 = np.zeros((1, w.n_orb), dtype=np.complex128)
        psi0[0, int(w.sites()[0])] = 1.0
    else:
        psi0 = w.psi0(device="cpu", n_state=1).numpy()
    K = len(oracle.cheb_coeff(w.rescale * w.dt))
    rowptr, col, val = oracle.build_csr(w.n_orb, on, hi, hj, hv)          # (re-built inside propagate; this one sizes nnz)
    nnz = int(rowptr[-1])

    def one(m):
        t0 = time.perf_counter()
        corr, norm2 = oracle.propagate(w.n_orb, on, hi, hj, hv, psi0, m, w.dt, w.rescale, form="csr")
        return time.perf_counter() - t0, corr

    t1, _ = one(1)
    m = max(1, min(int(seconds / max(t1, 1e-6)), 4096))
    times = []
    for it in range(warmup + steps):
        t, corr = one(m)
        if it >= warmup:
            times.append(t)
    t = max(times)
    value = m * (K - 1) * nnz / t
    return value, 1e3 * statistics.mean(times), f"1 state x {m} time steps ({m * (K - 1)} H-applications) of the full-size lattice, " \
        f"oracle row form incl. its CSR build", oracle.num_threads()


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import torch
    from paper_2509_26309_b200 import workloads as W  # noqa: F401
    w, cfg, ldos, n_state, n_step = workload_of(args.workload, "cpu", 0, args.n_step)
    value, ms, sample, cores = oracle_sample(w, args.workload, args.cpu_seconds, steps=max(1, args.steps), warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128", "data": "synthetic",
            "config": {"workload": w.name, "n_orb": w.n_orb, "nnz": w.nnz, "n_state": n_state, "n_step": n_step, "rescale": w.rescale,
                       "tau": math.pi},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------------
def main_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_26309_b200 import tbpm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the TBPM path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w, cfg, ldos, n_state, n_step = workload_of(args.workload, dev, rank, args.n_step)
    # each rank propagates its own batch of seeded states (sub-streams rank*n_state ...); H is replicated
    psi0 = None if ldos else w.psi0(device=dev, n_state=n_state, first_state=rank * n_state)
    sites = w.sites() if ldos else None
    K = len(tbpm.tbpm_cheb_coeff(w.rescale * w.dt))
    flags = 0

    pb, sb = tbpm.tbpm_build_bytes(w.n_orb, w.n_hop, w.onsite is not None, flags)
    corr = torch.zeros((n_state, n_step), dtype=torch.complex128, device=dev)
    norm2 = torch.zeros((n_state, n_step), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)          # > L2 (126 MB)
    state = {}

    def one_step(timers=None):
        flush.fill_(1)                                                     # evict L2 between iterations (untimed)
        if timers is not None:
            timers[0].record()
        H = tbpm.tbpm_build(w.n_orb, w.onsite, w.hop_i, w.hop_j, w.hop_val, flags)
        if "ws" not in state:
            state["ws"] = torch.empty(tbpm.tbpm_propagate_bytes(H, n_state), dtype=torch.uint8, device=dev)
        if timers is not None:
            timers[1].record()
        if ldos:
            lc, ln, _ = tbpm.tbpm_ldos(H, sites, n_step, w.dt, w.rescale, workspace=state["ws"])
            corr.copy_(lc); norm2.copy_(ln)
        else:
            tbpm.tbpm_propagate(H, psi0, n_step, w.dt, w.rescale, workspace=state["ws"], corr=corr, norm2=norm2)
        if timers is not None:
            timers[2].record()
        state["H"] = H
        return H

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        one_step()
    barrier()
    launches0 = tbpm.tbpm_total_launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    for i in range(args.steps):
        one_step(evs[i])
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = tbpm.tbpm_total_launch_count() - launches0
    step_ms = [e[0].elapsed_time(e[2]) for e in evs]                      # device time, build + propagate
    prop_ms = [e[1].elapsed_time(e[2]) for e in evs]
    total_ms = sum(step_ms)
    t = torch.tensor([total_ms, sum(prop_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, prop_total_ms = float(t[0]), float(t[1])
    H = state["H"]
    nnz = H.nnz
    happs = n_state * n_step * (K - 1)
    value = world * args.steps * happs * nnz / (total_ms * 1e-3)
    norm_dev = float((norm2 - 1).abs().max())

    # roofline of the dominant kernel (the fused Chebyshev term): algorithmic bytes per launch = matrix as stored + 3 vectors
    # of the tile the launch processes; average launch duration = propagate time / number of term launches
    tile = min(8, 1 << (n_state - 1).bit_length()) if not os.environ.get("TBPM_TILE") else int(os.environ["TBPM_TILE"])
    n_tile = -(-n_state // tile)
    term_launches = n_tile * n_step * (K - 1)
    avg_term_s = (prop_total_ms * 1e-3 / args.steps) / term_launches
    bytes_per_launch = H.matrix_bytes_per_term + 3 * 16 * w.n_orb * min(tile, n_state)
    peak, peak_src = load_peaks()
    achieved = bytes_per_launch / avg_term_s / 1e9
    roofline = {"bound": "hbm", "kernel": "k_term_ph (fused Chebyshev term, term_ph.cuh)", "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic(w.name, K), "traffic_source": NCU_TRAFFIC_SRC,
                "peak_source": peak_src, "bytes_per_launch": bytes_per_launch,
                "avg_launch_us": avg_term_s * 1e6, "launches_per_step": term_launches,
                "counted_csr_gbs": (8 * (w.n_orb + 1) + 20 * nnz + 48 * w.n_orb * min(tile, n_state)) / avg_term_s / 1e9,
                "frac_of_nominal_8000": achieved / 8000.0,
                "note": "avg launch = CUDA-event time of tbpm_propagate / term launches (includes the <1% of tiny kernels)"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128", "data": "synthetic",
            "config": {"workload": w.name, "n_orb": w.n_orb, "nnz": nnz, "n_state": n_state, "n_step": n_step, "K": K, "rescale": w.rescale,
                       "tau": math.pi, "tile": tile, "n_table": H.n_table, "matrix_bytes_per_term": H.matrix_bytes_per_term,
                       "l2": "256 MB flush between iterations; working set > L2", "ldos": ldos,
                       "parallelism": f"replicas x{world}: each rank its own {n_state} states"},
            "ms_build": sum(e[0].elapsed_time(e[1]) for e in evs) / args.steps, "ms_propagate": prop_total_ms / args.steps,
            "h_apps_per_s": world * args.steps * happs / (total_ms * 1e-3), "ms_per_time_step": prop_total_ms / args.steps / n_step,
            "max_norm_dev": norm_dev, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}
    if args.n_step:
        line["config"]["n_step_override"] = args.n_step

    # end to end through the C ABI with HOST buffers: H2D of the hop list and psi0, build, propagate, D2H of corr/norm2
    if not args.no_e2e and not ldos:
        hw = {k: getattr(w, k).cpu().pin_memory() for k in ("hop_i", "hop_j", "hop_val")}
        hon = None if w.onsite is None else w.onsite.cpu().pin_memory()
        hpsi = psi0.cpu().pin_memory()
        hcorr = torch.zeros((n_state, n_step), dtype=torch.complex128).pin_memory()
        hnorm = torch.zeros((n_state, n_step), dtype=torch.float64).pin_memory()
        state.clear()
        arena = torch.empty(tbpm.tbpm_corr_host_bytes(w.n_orb, w.n_hop, hon is not None, n_state, n_step, flags), dtype=torch.uint8, device=dev)
        up = down = 0
        e2e_t = []
        for i in range(1 + max(1, min(args.steps, 2))):
            barrier()
            t0 = time.perf_counter()
            up, down = tbpm.tbpm_corr_host(w.n_orb, hon, hw["hop_i"], hw["hop_j"], hw["hop_val"], hpsi, n_step, w.dt, w.rescale, arena,
                                           hcorr, hnorm, flags)
            if i > 0:
                e2e_t.append(time.perf_counter() - t0)
        te = torch.tensor([sum(e2e_t)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        line["e2e"] = {"value": world * len(e2e_t) * happs * nnz / float(te[0]), "unit": UNIT, "h2d_bytes_per_step": int(up),
                       "d2h_bytes_per_step": int(down), "ms_per_step": 1e3 * float(te[0]) / len(e2e_t),
                       "max_abs_diff_vs_device_path": float((hcorr.to(dev) - corr).abs().max())}
        del arena

    if rank == 0 and not args.no_cpu_baseline:
        v, ms, sample, cores = oracle_sample(w, args.workload, args.cpu_seconds)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse_args()
    sys.exit(main_reference(a) if a.impl == "reference" else main_ours(a))
