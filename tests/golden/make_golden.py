#!/usr/bin/env python
"""Write stored oracle outputs for the long propagations no test can afford to recompute.

    python tests/golden/make_golden.py --config 2                 # full length (15 cm, 3000 RK4IP steps, ~1 h CPU)
    python tests/golden/make_golden.py --config 3 --length 0.02   # first 2 cm of config 3 (200 steps, ~20 min CPU)

Calls only ``oracle/`` (fp64 RK4IP, oracle O3) and the seeded input generators; never the CUDA path.  The launch
field is rounded to complex64 first, exactly what the GPU tests feed the library.  Output: a text file with the
propagated field sampled every ``--stride``-th time sample for every mode (columns: mode, sample, re, im) and a
header holding the run parameters and a checksum of the inputs, which the test verifies before comparing.
"""
import argparse
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import gmmnlse_oracle as O                      # noqa: E402
from paper_1708_05324_b200 import workloads as W           # noqa: E402


def input_checksum(w, A_in):
    h = hashlib.sha256()
    for a in (A_in, w.S, w.beta, w.h_R if w.h_R is not None else np.zeros(1)):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()[:32]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--length", type=float, default=None, help="propagation length in m (default: the full L)")
    ap.add_argument("--stride", type=int, default=8)
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    w = W.make_config(args.config)
    L = w.L if args.length is None else args.length
    steps = int(round(L / w.dz))
    A_in = w.A0.astype(np.complex64).astype(np.complex128)
    omega = O.omega_grid(w.N, w.dt)
    D = O.dispersion_operator(w.beta, omega)
    nl = lambda X: O.nonlinear_op_freq(X, w.S, w.kappa, omega, w.omega0, w.f_R, w.h_R, w.dt, w.shock)
    At = O.to_freq(A_in)
    t0 = time.time()
    for i in range(steps):
        At = O.rk4ip_step(At, w.dz, D, nl)
        if (i + 1) % 100 == 0:
            print(f"step {i + 1}/{steps}  {time.time() - t0:.0f} s", flush=True)
    out = O.to_time(At)
    name = args.out or os.path.join(os.path.dirname(os.path.abspath(__file__)),
                                    f"config{args.config}_rk4ip_{steps}steps.txt")
    idx = np.arange(0, w.N, args.stride)
    rows = [(p, n, out[p, n].real, out[p, n].imag) for p in range(w.P) for n in idx]
    pn = float(O.photon_number(out, w.dt, w.omega0) / O.photon_number(A_in, w.dt, w.omega0))
    header = (f"oracle RK4IP (oracle/gmmnlse_oracle.py rk4ip_step), BASELINE.json config {args.config}\n"
              f"L_m={float(L)!r} dz_m={float(w.dz)!r} steps={steps} P={w.P} N={w.N} stride={args.stride}\n"
              f"input_sha256_32={input_checksum(w, A_in)}\n"
              f"energy_in={float(O.energy(A_in, w.dt))!r} energy_out={float(O.energy(out, w.dt))!r}\n"
              f"photon_number_ratio={pn!r}\n"
              "columns: mode sample re im")
    np.savetxt(name, np.array(rows), fmt=["%d", "%d", "%.17e", "%.17e"], header=header)
    print("wrote", name, f"({time.time() - t0:.0f} s)")


if __name__ == "__main__":
    main()
