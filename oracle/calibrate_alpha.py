"""Writes the MLIP energy scales alpha used by lsd_inputs.workloads.ALPHA.

Rule: on a thermalised reference configuration (500 prior-only ABOBA steps from the seeded start, Maxwell-Boltzmann
momenta) alpha = 0.10 * RMS(F_prior) / RMS(F_NN at alpha = 1).  Calls only oracle/ (and the input generators).
Scaled-down boxes with the same density and local structure are used for cfg4/cfg5 (the ratio is intensive).

    python -m oracle.calibrate_alpha          # prints the table to paste into lsd_inputs/workloads.py
"""
import dataclasses
import sys

import numpy as np

import lsd_inputs as L
import oracle
from lsd_inputs.workloads import Potential

CASES = [("cfg2", {}), ("cfg3", {"n_grid": 6}), ("cfg4", {"n_atoms": 1500}), ("cfg5", {"cells": (6, 6, 6)})]


def main():
    for name, kw in CASES:
        w = L.make_workload(name, **kw)
        prior = Potential(w.target.pair, w.target.use_bonded, None)
        p0 = oracle.initial_momenta(w)
        th = oracle.run_aboba(w, prior, w.q0, p0, 500, keep_traj=False)
        q = th["q"]
        Fp = oracle.energy_forces(w, prior, q)[1]
        rms_p = np.sqrt((Fp**2).mean())
        for role in ("target", "draft"):
            pot = getattr(w, role)
            if pot.mlip is None:
                continue
            m1 = dataclasses.replace(pot.mlip, alpha=1.0)
            Fn = oracle.mlip_energy_forces(w, m1, q)[1]
            rms_n = np.sqrt((Fn**2).mean())
            print(f'    ("{name}", "{role}"): {0.10 * rms_p / rms_n:.6e},   # rms prior {rms_p:.4f} eV/A, rms NN(alpha=1) {rms_n:.4f}')
            sys.stdout.flush()


if __name__ == "__main__":
    main()
