#!/usr/bin/env python
"""Write stored oracle outputs for the long propagations no test can afford to recompute.

    python tests/golden/make_golden.py --config 2                      # full length (15 cm, 3000 RK4IP steps)
    python tests/golden/make_golden.py --config 3                      # full length (1 m, 10^4 RK4IP steps)
    python tests/golden/make_golden.py --config 3 --integrator mpa     # the same with the oracle's plain MPA (O4)
    python tests/golden/make_golden.py --config 3 --length 0.02 --dz-div 4   # converged reference: RK4IP at dz/4

Calls only ``oracle/`` (fp64 RK4IP = O3, plain MPA = O4) and the seeded input generators; never the CUDA path.  The
launch field is rounded to complex64 first, exactly what the GPU tests feed the library.  Output: the WHOLE propagated
field ``[P][N]`` complex128 as ``<name>.npy`` and the run parameters, a fingerprint of the inputs and the oracle's own
conserved-quantity ratio as ``<name>.json``, which the tests verify before comparing every element.

Long runs checkpoint their state every ``--checkpoint-every`` steps into ``--work-dir`` (default: the system temporary
directory) and resume from there when re-run with the same arguments.
"""
import argparse
import json
import os
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import gmmnlse_oracle as O                      # noqa: E402
from paper_1708_05324_b200 import workloads as W           # noqa: E402

GOLDEN_DIR = os.path.dirname(os.path.abspath(__file__))


def input_fingerprint(w, A_in):
    """A few sums of the inputs (launch field, S, beta, h_R).  Compared with rtol 1e-9, not bit for bit: the
    quadrature behind S goes through BLAS, whose summation order differs between hosts in the last bits."""
    h = w.h_R if w.h_R is not None else np.zeros(1)
    ws = 1.0 + np.arange(w.S.size, dtype=np.float64).reshape(w.S.shape) / w.S.size      # position-sensitive weights,
    wa = 1.0 + np.arange(A_in.size, dtype=np.float64).reshape(A_in.shape) / A_in.size   # sums of magnitudes: no
    wh = 1.0 + np.arange(h.size, dtype=np.float64) / h.size                             # cancellation
    return {"fp_A": float(np.sum(np.abs(A_in) ** 2 * wa)), "fp_S": float(np.sum(np.abs(w.S) * ws)),
            "fp_beta": float(np.sum(np.abs(w.beta))), "fp_h": float(np.sum(np.abs(h) * wh))}


def fingerprint_matches(meta, w, A_in, rtol=1e-9):
    fp = input_fingerprint(w, A_in)
    return all(k in meta and abs(float(meta[k]) - v) <= rtol * max(abs(v), 1e-300) for k, v in fp.items())


def golden_name(config, integrator, steps, dz_div=1):
    return f"config{config}_{integrator}_{steps}steps" + (f"_dzdiv{dz_div}" if dz_div != 1 else "")


def load_golden(name):
    """(meta dict, field [P][N] complex128) of a stored run, or None if it was not generated."""
    base = os.path.join(GOLDEN_DIR, name)
    if not (os.path.exists(base + ".npy") and os.path.exists(base + ".json")):
        return None
    with open(base + ".json") as fh:
        meta = json.load(fh)
    return meta, np.load(base + ".npy")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--length", type=float, default=None, help="propagation length in m (default: the full L)")
    ap.add_argument("--dz-div", type=int, default=1, help="integrate with dz / this (converged references)")
    ap.add_argument("--integrator", default="rk4ip", choices=["rk4ip", "mpa"],
                    help="oracle O3 (RK4IP, default) or O4 (plain MPA with the configuration's M and tol)")
    ap.add_argument("--checkpoint-every", type=int, default=200, help="small steps between checkpoints")
    ap.add_argument("--work-dir", default=None)
    ap.add_argument("--out-dir", default=GOLDEN_DIR)
    args = ap.parse_args()
    w = W.make_config(args.config)
    L = w.L if args.length is None else args.length
    dz = w.dz / args.dz_div
    steps_cfg = int(round(L / w.dz))            # length in units of the configuration's own dz (names the file)
    steps = steps_cfg * args.dz_div
    A_in = w.A0.astype(np.complex64).astype(np.complex128)
    omega = O.omega_grid(w.N, w.dt)
    D = O.dispersion_operator(w.beta, omega)
    nl = lambda X: O.nonlinear_op_freq(X, w.S, w.kappa, omega, w.omega0, w.f_R, w.h_R, w.dt, w.shock)
    name = golden_name(args.config, args.integrator, steps_cfg, args.dz_div)
    work = args.work_dir or tempfile.gettempdir()
    os.makedirs(work, exist_ok=True)
    ck = os.path.join(work, name + ".ckpt.npz")
    fp = input_fingerprint(w, A_in)
    # ---- state: the frequency-domain field after `done` small steps (+ MPA counters) ----
    At, done, n_large, n_iter, n_noconv, elapsed = O.to_freq(A_in), 0, 0, 0, 0, 0.0
    if os.path.exists(ck):
        z = np.load(ck)
        if abs(float(z["fp_A"]) - fp["fp_A"]) <= 1e-9 * fp["fp_A"] and int(z["steps"]) == steps:
            At, done = z["At"], int(z["done"])
            n_large, n_iter, n_noconv, elapsed = int(z["n_large"]), int(z["n_iter"]), int(z["n_noconv"]), float(z["elapsed"])
            print(f"resuming {name} at step {done}/{steps}", flush=True)
    t0 = time.time() - elapsed

    def checkpoint():
        tmp = ck + ".tmp.npz"
        np.savez(tmp, At=At, done=done, steps=steps, n_large=n_large, n_iter=n_iter, n_noconv=n_noconv,
                 elapsed=time.time() - t0, fp_A=fp["fp_A"])
        os.replace(tmp, ck)

    last_ck = done
    if args.integrator == "mpa":
        # the loop of oracle.mpa_propagate, one large step at a time so that the state can be checkpointed
        K = 1j * w.kappa * (1.0 + omega / w.omega0 if w.shock else np.ones_like(omega))
        nl_time = lambda A: O.nonlinear_term(A, w.S, w.f_R, w.h_R, w.dt)
        while done < steps:
            Mc = min(w.M, steps - done)
            At, it, _, conv = O.mpa_large_step(At, Mc, dz, D, nl_time, K, w.tol)
            done += Mc
            n_large += 1
            n_iter += it
            n_noconv += 0 if conv else 1
            if done - last_ck >= args.checkpoint_every or done == steps:
                checkpoint()
                last_ck = done
                print(f"step {done}/{steps}  {time.time() - t0:.0f} s  iterations {n_iter}", flush=True)
    else:
        while done < steps:
            At = O.rk4ip_step(At, dz, D, nl)
            done += 1
            if done - last_ck >= args.checkpoint_every or done == steps:
                checkpoint()
                last_ck = done
                print(f"step {done}/{steps}  {time.time() - t0:.0f} s", flush=True)
    out = O.to_time(At)
    which = "RK4IP (oracle/gmmnlse_oracle.py rk4ip_step)" if args.integrator == "rk4ip" else \
        "plain MPA (oracle/gmmnlse_oracle.py mpa_large_step)"
    meta = {"what": f"oracle {which}, BASELINE.json config {args.config}",
            "command": "python tests/golden/make_golden.py " + " ".join(sys.argv[1:]),
            "config": args.config, "integrator": args.integrator, "L_m": float(L), "dz_m": float(dz),
            "dz_div": args.dz_div, "steps": steps, "P": w.P, "N": w.N,
            "energy_in": float(O.energy(A_in, w.dt)), "energy_out": float(O.energy(out, w.dt)),
            "photon_number_ratio": float(O.photon_number(out, w.dt, w.omega0) / O.photon_number(A_in, w.dt, w.omega0)),
            "cpu_seconds_wall": round(time.time() - t0, 1)}
    if args.integrator == "mpa":
        meta.update(M=w.M, tol=float(w.tol), large_steps=n_large, iterations=n_iter, not_converged=n_noconv)
    meta.update(fp)
    base = os.path.join(args.out_dir, name)
    np.save(base + ".npy", out.astype(np.complex128))
    with open(base + ".json", "w") as fh:
        json.dump(meta, fh, indent=1)
        fh.write("\n")
    print("wrote", base + ".npy", f"({time.time() - t0:.0f} s)")


if __name__ == "__main__":
    main()
