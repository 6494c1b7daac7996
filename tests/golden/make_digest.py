"""Writes the full-size oracle digests under tests/golden/ (test infrastructure, NOT the product; sits beside the
files it writes).

A full fp64 oracle solve of a 512^3 network takes about an hour of host time, too long for the GPU test run, so it
is done once, here, and what the GPU parity test needs is stored (SURVEY.md 8(d) option (c); BASELINE.json north_star
"a 512^3 correlated network ... matching the oracle within the stated tolerances"):

    tests/golden/<name>_digest.json   input SHA-256, class counts, iterations, true residuals, Q_in, Q_out, G_eff,
                                      the n_a - 1 plane fluxes, the oracle's own error estimate, host timings
    tests/golden/<name>_P_sub8.npy    the oracle's pressures on every 8th node per axis, offset 4 (fp64, 2 MB)

Every number comes from oracle/ (pn_oracle.c through c_oracle.py) applied to the seeded input recipe
(paper_1908_03301_b200/inputs.py holds generators only); nothing here touches the CUDA path.

Steps per network and direction (SURVEY.md 8(c) consequence (iii)): solve from zero to tol 1e-12; carry that iterate
on to tol 1e-13 (same loop with its true-residual restarts, `P_start`); the difference between the two on ALL nodes
is the oracle's own error estimate, published beside the values.

    python tests/golden/make_digest.py cfg4            # 512^3, x          (about an hour on 8 cores)
    python tests/golden/make_digest.py cfg5            # 512^3, x and z
    python tests/golden/make_digest.py cfg4 --n 64     # a small sibling (used by the CPU tests to check this script)
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

from oracle import c_oracle                                   # noqa: E402
from paper_1908_03301_b200 import inputs                      # noqa: E402  (seeded generators only)

STRIDE, OFFSET = 8, 4


def sub_sample(P: np.ndarray) -> np.ndarray:
    """Every 8th node per axis starting at 4 (axes shorter than 5 nodes: every node)."""
    sl = tuple(slice(OFFSET, None, STRIDE) if n > OFFSET else slice(None) for n in P.shape)
    return np.ascontiguousarray(P[sl])


def plane_fluxes(net, P: np.ndarray, direction: int) -> np.ndarray:
    """Total flow through each of the n_a - 1 planes of bonds normal to the solve axis (eq.(4))."""
    g = (net.gx, net.gy, net.gz)[direction].reshape(net.nz, net.ny, net.nx)
    ax = 2 - direction
    n_a = P.shape[ax]
    out = np.empty(n_a - 1)
    for c in range(n_a - 1):
        s0 = [slice(None)] * 3
        s1 = [slice(None)] * 3
        s0[ax], s1[ax] = c, c + 1
        out[c] = np.sum(g[tuple(s0)].astype(np.float64) * (P[tuple(s0)] - P[tuple(s1)]))
    return out


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def digest(net, direction: int, threads: int, log=print) -> tuple:
    t0 = time.time()
    a = c_oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-12, threads=threads)
    log(f"  tol 1e-12: {a.iterations} iterations, true residual {a.rel_residual:.3e}, {time.time() - t0:.0f} s")
    t1 = time.time()
    b = c_oracle.solve(net.nx, net.ny, net.nz, net.gx, net.gy, net.gz, direction, 1e-13, threads=threads,
                       P_start=a.P)
    log(f"  tol 1e-13: +{b.iterations} iterations, true residual {b.rel_residual:.3e}, {time.time() - t1:.0f} s")
    assert np.array_equal(a.classes, b.classes)
    pf = plane_fluxes(net, b.P, direction)
    d = {
        "network": net.name, "nx": net.nx, "ny": net.ny, "nz": net.nz, "direction": direction,
        "input_sha256": net.sha256(),
        "n_solved": b.n_solved, "n_inlet_only": b.n_inlet_only, "n_outlet_only": b.n_outlet_only,
        "n_floating": b.n_floating, "nnz": b.nnz,
        "status_1e12": a.status, "status_floor": b.status,
        "iterations_to_1e12": a.iterations, "restarts_to_1e12": a.restarts,
        "iterations_1e12_to_floor": b.iterations,
        # first iteration of the zero-start PCG whose recursive ||r||/||b|| <= 1e-k (k = list index)
        "iterations_at_decade": list(a.it_decade),
        "true_residual_1e12": a.rel_residual, "true_residual_floor": b.rel_residual,
        "q_in": b.q_in, "q_out": b.q_out, "g_eff": b.g_eff, "k_eff": b.k_eff,
        "g_eff_1e12": a.g_eff,
        "plane_fluxes": [float(v) for v in pf],
        # the oracle's own error estimate: |P(1e-12) - P(floor)| over ALL nodes, and the same on G_eff
        "error_estimate_P_linf": float(np.max(np.abs(a.P - b.P))),
        "error_estimate_g_eff_rel": abs(a.g_eff - b.g_eff) / abs(b.g_eff) if b.g_eff else 0.0,
        "sub_sample": {"stride": STRIDE, "offset": OFFSET, "shape": list(sub_sample(b.P).shape)},
        "host": {"cpu": cpu_model(), "threads": a.threads, "t_label_s": a.t_label, "t_assemble_s": a.t_assemble,
                 "t_pcg_to_1e12_s": a.t_pcg, "s_per_iteration": a.t_pcg / max(a.iterations, 1),
                 "t_pcg_1e12_to_floor_s": b.t_pcg},
    }
    return d, sub_sample(b.P)


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("config", choices=["cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--n", type=int, default=0, help="edge length of a scaled-down sibling (default: full size)")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--out", default=HERE)
    args = ap.parse_args(argv)
    gen = {"cfg2": inputs.cfg2_fbm_2d, "cfg3": inputs.cfg3_percolation_3d, "cfg4": inputs.cfg4_fbm_cut_3d,
           "cfg5": inputs.cfg5_stratified_3d}[args.config]
    t = time.time()
    net = (gen(args.n, args.n) if args.config == "cfg2" else gen(args.n, args.n, args.n)) if args.n else gen()
    print(f"{net.name}: generated in {time.time() - t:.0f} s, sha256 {net.sha256()}", flush=True)
    os.makedirs(args.out, exist_ok=True)
    for direction in net.directions:
        print(f" direction {direction}", flush=True)
        d, sub = digest(net, direction, args.threads, log=lambda s: print(s, flush=True))
        edge = max(net.nx, net.ny, net.nz)
        stem = os.path.join(args.out, f"{args.config}_{edge}_{'xyz'[direction]}")
        np.save(stem + "_P_sub8.npy", sub)
        with open(stem + "_digest.json", "w") as f:
            json.dump(d, f, indent=1)
        print(f"  wrote {stem}_digest.json, G_eff {d['g_eff']!r}, error estimate {d['error_estimate_P_linf']:.2e}",
              flush=True)


if __name__ == "__main__":
    main()
