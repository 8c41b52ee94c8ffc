"""Run config C2 of BASELINE.json end to end: N = 32768 equal-mass Plummer sphere, eps = 1e-4,
4th-order Hermite with block time steps (eta = 0.01, power-of-two steps), driven through the
GRAPE-6 calling sequence of libg6b200 (Fig. 1).

    python -m paper_0902_4463_b200.hermite_run [--n 32768] [--t-end 1.0] [--eta 0.01] [--newton 1] [--driver host|device]

Prints one JSON line: block-step statistics, the n_i histogram, wall-clock rates and (with
--state-out) writes the final state for an independent energy check.  The energy itself is the
checker's business (tests/ and the oracle), not this module's.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

from . import build, g6, inputs


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=None)
    ap.add_argument("--t-end", type=float, default=1.0)
    ap.add_argument("--eta", type=float, default=0.01)
    ap.add_argument("--newton", type=int, default=None)
    ap.add_argument("--driver", default="host", choices=["host", "device"],
                    help="host: g6h_* (host corrector, GRAPE-6 calling sequence); device: g6hd_* (corrector and block selection on the GPU)")
    ap.add_argument("--state-out", default=None, help=".npz file for the initial and final state")
    args = ap.parse_args()
    build.build()
    x, v, m, eps2 = inputs.config("C2", n=args.n)
    g6.g6_open(0)
    if args.newton is not None:
        g6.g6x_set_option(0, "newton", args.newton)
    t0 = time.perf_counter()
    h = (g6.HermiteDev if args.driver == "device" else g6.Hermite)(0, x, v, m, eps2, args.eta)
    t_init = time.perf_counter() - t0
    h.evolve(args.t_end)
    x1, v1 = h.state()
    st = h.stats()
    h.close()
    g6.g6_close(0)
    hist = [int(c) for c in st["ni_hist_log2"][:24]]
    st.setdefault("wall_force_s", float("nan")); st.setdefault("force_wall_s_log2", np.zeros(64))
    out = {"config": "C2", "driver": args.driver, "n": len(m), "eps2": eps2, "eta": args.eta, "t_end": st["t"],
           "block_steps": st["n_block_steps"], "particle_steps": st["n_particle_steps"],
           "mean_block_size": st["n_particle_steps"] / max(1, st["n_block_steps"]),
           "interactions": st["interactions"], "dt_min": st["dt_min"],
           "wall_s": st["wall_s"], "wall_force_calls_s": st["wall_force_s"], "init_s": t_init,
           "block_steps_per_s": st["n_block_steps"] / max(st["wall_s"], 1e-9),
           "interactions_per_s": st["interactions"] / max(st["wall_s"], 1e-9),
           "gflops_60": 60 * st["interactions"] / max(st["wall_s"], 1e-9) / 1e9,
           "ni_hist_log2": hist, "force_wall_s_log2": [round(float(w), 4) for w in st["force_wall_s_log2"][:24]]}
    if args.state_out:
        np.savez(args.state_out, x0=x, v0=v, m=m, x1=x1, v1=v1, eps2=eps2)
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
