"""Writes tests/golden/cfg4_step1.npz: the CPU oracle's state after ONE RK4 step of BASELINE config 4
(2^11 x 2^11 decaying turbulence, chi = 128, chi_work = 256, Re = 1e6, dt = 0.1/2^10, eps = 0).

    python tests/golden/make_cfg4_step.py            # from the repo root; ~10-25 min on 8-16 host cores

Imports ONLY oracle/ and qtt_inputs/ (no CUDA path): the stored values are the oracle's.  The GPU parity test
tests/test_gpu_parity.py::test_config4_full_step_matches_stored_oracle recomputes the input cores with the oracle's
from_dense (seconds), feeds them to qtt_rk4_step and compares dense fields, bonds and Schmidt spectra.
Stored: the output cores u1_i_k (fp64) and the oracle's Schmidt values of the output per bond (sv1_i_k).
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import qtt_inputs as I  # noqa: E402
from oracle import qtt_oracle as O  # noqa: E402


def main():
    cfg = 4
    c = I.CONFIGS[cfg]
    n, chi = c["n"], c["chi"]
    dx = 1.0 / (1 << n)
    ux, uy = I.config_fields(cfg)
    t0 = time.perf_counter()
    U = [O.from_dense(ux, chi), O.from_dense(uy, chi)]
    ops = (O.mpo_d1(n, dx), O.mpo_d2(n, dx), O.mpo_laplacian(n, dx))
    print(f"from_dense {time.perf_counter() - t0:.1f} s", flush=True)
    t0 = time.perf_counter()
    U1 = O.rk4_step(U, *ops, c["Re"], c["dt"], chi)
    print(f"oracle rk4_step {time.perf_counter() - t0:.1f} s", flush=True)
    out = {"n": n, "chi": chi, "Re": c["Re"], "dt": c["dt"]}
    for i in range(2):
        for k in range(n):
            out[f"u1_{i}_{k}"] = U1[i][k]
        sv = O.schmidt_values(U1[i])
        for k in range(1, n):
            out[f"sv1_{i}_{k}"] = sv[k]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg4_step1.npz")
    np.savez_compressed(path, **out)
    print("wrote", path, os.path.getsize(path), "bytes", flush=True)


if __name__ == "__main__":
    main()
