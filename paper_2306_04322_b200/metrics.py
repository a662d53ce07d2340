"""Harness-side metrics of the paper (no method arithmetic of the stepping path; numpy only).

eq22: the paper's normalised squared L2 error (Eq. 22; no square root),
      E_phi = sum_x (phi - phi_ref)^2 / sum_x phi_ref^2,  phi = c or phi = sum_i eta_i.
The oracle states the same definition independently (oracle/pfo.c: pfo_error_eq22, pinned by closed forms);
tests/test_oracle_steps.py checks this function against it.
"""
import numpy as np


def eq22(phi, ref) -> float:
    phi = np.asarray(phi, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    return float(np.sum((phi - ref) ** 2) / np.sum(ref ** 2))


def eq22_percent(phi, ref) -> float:
    return 100.0 * eq22(phi, ref)
