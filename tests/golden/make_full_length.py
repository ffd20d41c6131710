#!/usr/bin/env python
"""Writes tests/golden/corr_full_cfg*.txt: FULL-LENGTH oracle runs of BASELINE.json's configs (parity protocol (6) of
SURVEY.md section 8(d): "full-length oracle runs ... done once in the background and cached to disk keyed by (config, seed)").

It calls ONLY oracle/ (the CPU statement of PAPER.md:437-443, OpenMP row form, itself pinned to the serial hop form by
tests/test_oracle_pins.py::test_row_form_matches_hop_form) and the seeded input generators; nothing here touches the
CUDA library.  One file per (config, state): every time step's corr and norm2 at %.17e (round-trips a double).

    python tests/golden/make_full_length.py 2 3 4 5        # about 1.5 h on 8 host cores for all four
States: config 2 all four; configs 3 / 4 / 5 one seeded state each (index below), full n_step (1024 / 2048 / 1024).
"""
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np

import oracle
from paper_2509_26309_b200 import workloads as W

STATES = {1: [0], 2: [0, 1, 2, 3], 3: [0], 4: [3], 5: [5]}
HERE = os.path.dirname(os.path.abspath(__file__))


def path(cfg: int, state: int) -> str:
    return os.path.join(HERE, f"corr_full_cfg{cfg}_state{state}.txt")


def main(cfgs):
    for cfg in cfgs:
        w = W.make_workload(cfg)
        hi, hj, hv = w.hop_i.numpy(), w.hop_j.numpy(), w.hop_val.numpy()
        on = None if w.onsite is None else w.onsite.numpy()
        for s in STATES[cfg]:
            if os.path.exists(path(cfg, s)):
                continue
            psi0 = W.random_phase_state(w.n_orb, s, w.seed).numpy()[None, :]
            t0 = time.time()
            corr, norm2 = oracle.propagate(w.n_orb, on, hi, hj, hv, psi0, w.n_step, w.dt, w.rescale, form="csr")
            with open(path(cfg, s), "w") as f:
                f.write(f"# Full-length ORACLE run (oracle.propagate, form=csr) of BASELINE.json:configs[{cfg - 1}] = {w.name}\n")
                f.write(f"# state {s} of the seeded random-phase stream (seed {w.seed}), n_orb {w.n_orb}, n_step {w.n_step}, rescale {w.rescale}, tau = pi\n")
                f.write("# written by tests/golden/make_full_length.py, which calls only oracle/ and the input generators\n")
                f.write("# step  Re corr  Im corr  norm2      (entry n is t = (n+1) dt)\n")
                for n in range(w.n_step):
                    f.write(f"{n} {corr[0, n].real:.17e} {corr[0, n].imag:.17e} {norm2[0, n]:.17e}\n")
            print(f"cfg{cfg} state {s}: {time.time() - t0:.0f} s, max|norm2-1| = {np.abs(norm2 - 1).max():.2e}", flush=True)


def load(cfg: int, state: int):
    a = np.loadtxt(path(cfg, state))
    return a[:, 1] + 1j * a[:, 2], a[:, 3]


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [2, 3, 4, 5])
