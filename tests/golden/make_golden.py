"""Writes tests/golden/obs_cfg<i>.txt: the seeded synthetic observation of each
BASELINE.json workload, D_j = M_j(theta_true) (1 + 0.02 eps_j), err_j = 0.02 M_j.

Calls ONLY the oracle (oracle/) and the input generators (workloads/); nothing
here ever comes from the CUDA path.  Usage:

    python tests/golden/make_golden.py [config indices ...]      # default: 0 1 2 3

Config 4 re-uses config 3's tables, grid and observation.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads as W  # noqa: E402
from workloads.generate import noise_draw  # noqa: E402


def main(indices):
    for i in indices:
        cfg = W.get_config(i)
        wl = W.make_workload(i, batch=1)
        theta = W.true_params(cfg)[None, :]
        r = oracle.forward_workload(wl, params=theta, want_spectra=True, want_logl=False)
        M = r["spectra"][0]
        eps = noise_draw(cfg)
        D = M * (1.0 + 0.02 * eps)
        err = 0.02 * M
        path = os.path.join(W.golden_dir(), f"obs_cfg{i}.txt")
        with open(path, "w") as fh:
            fh.write(f"# Synthetic observation for BASELINE.json configs[{i}] ({cfg.name}).\n")
            fh.write("# D_j = M_j(theta_true) (1 + 0.02 eps_j), err_j = 0.02 M_j; M from oracle/helios_oracle.c\n")
            fh.write("# (fp64), theta_true = workloads.true_params, eps = workloads.generate.noise_draw.\n")
            fh.write("# Written by tests/golden/make_golden.py; stands in for the SpeX/ISAAC spectra of PAPER.md:443-457.\n")
            fh.write("# theta_true = " + " ".join(repr(float(v)) for v in theta[0]) + "\n")
            fh.write("# columns: D_j  err_j   [erg s^-1 cm^-2 (cm^-1)^-1]\n")
            for d, e in zip(D, err):
                fh.write(f"{d!r} {e!r}\n".replace("np.float64(", "").replace(")", ""))
        print("wrote", path, "clamped", r["n_clamped"])


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [0, 1, 2, 3])
