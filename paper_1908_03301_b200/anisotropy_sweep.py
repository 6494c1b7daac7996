#!/usr/bin/env python
"""Permeability anisotropy K_x / K_y of 2D networks with an anisotropic FBM conductance field
(eq.(2); the experiment of Fig.10).

    python -m paper_1908_03301_b200.anisotropy_sweep [--n 1024] [--H 0.75 0.35] [--ratios 0.25 0.5 1 2 4]
                                                     [--realisations 4] [--sigma 1.0] [--no-flux] [--tol 1e-10]

For every Hurst exponent H and every ratio beta_x / beta_y it generates `realisations` seeded networks
(inputs.aniso_fbm_2d), solves each one twice through the C ABI (pressure drop along x, then along y; lateral
faces periodic as in the paper, unless --no-flux) and prints one JSON line with the mean and the standard
deviation of K_x / K_y.  The paper gives only the RANGES it read off its Fig.10 (H = 0.75: 0.6 .. 1.6;
H = 0.35: 0.5 .. about 2.5) and neither the beta ratios, the network size nor the conductance map, so this
reproduces the experiment's shape, not its numbers.  Inputs are synthetic and seeded; nothing is read from disk.
Needs a CUDA device (there is no CPU fallback).
"""
from __future__ import annotations

import argparse
import json
import math
import time


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=1024)
    ap.add_argument("--H", type=float, nargs="+", default=[0.75, 0.35])
    ap.add_argument("--ratios", type=float, nargs="+", default=[0.25, 0.5, 1.0, 2.0, 4.0])
    ap.add_argument("--realisations", type=int, default=4)
    ap.add_argument("--sigma", type=float, default=1.0)
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--no-flux", action="store_true", help="no-flux lateral faces instead of the paper's periodic ones")
    ap.add_argument("--seed", type=int, default=100)
    args = ap.parse_args()

    from . import build, inputs, pn
    build.build()
    h = pn.Network(args.n, args.n, 1)
    h.set_option(pn.PN_OPT_LATERAL, 0 if args.no_flux else 1)
    for H in args.H:
        for ratio in args.ratios:
            vals, iters, t0 = [], 0, time.perf_counter()
            for rep in range(args.realisations):
                # beta_x * beta_y = 1 keeps the geometric-mean correlation length fixed while the ratio changes
                bx, by = math.sqrt(ratio), 1.0 / math.sqrt(ratio)
                net = inputs.aniso_fbm_2d(args.n, args.n, args.seed + rep, H, bx, by, args.sigma)
                h.set_conductances(net.gx, net.gy, None)
                k = []
                for d in (0, 1):
                    info = h.solve(d, args.tol, accept=(pn.PN_OK,))
                    iters += info.inner_iters
                    k.append(h.flux()[3])
                vals.append(k[0] / k[1])
            mean = sum(vals) / len(vals)
            std = math.sqrt(sum((v - mean) ** 2 for v in vals) / max(len(vals) - 1, 1))
            print(json.dumps({"H": H, "beta_x_over_beta_y": ratio, "n": args.n, "sigma": args.sigma,
                              "lateral": "no-flux" if args.no_flux else "periodic", "realisations": args.realisations,
                              "Kx_over_Ky_mean": mean, "Kx_over_Ky_std": std, "values": vals,
                              "inner_iters": iters, "wall_s": round(time.perf_counter() - t0, 2)}), flush=True)
    h.close()


if __name__ == "__main__":
    main()
