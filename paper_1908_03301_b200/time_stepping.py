#!/usr/bin/env python
"""A sequence of re-solves of one network whose conductances drift from step to step (a flow or transport
process "may take thousands of time steps").

    python -m paper_1908_03301_b200.time_stepping [--workload cfg4] [--n 512] [--steps 10] [--fraction 0.01]
                                                  [--eps 0.05] [--tol 1e-10] [--flip 0]

Step 0 is the cold solve (pn_set_conductances + pn_solve).  Every later step changes a random `fraction` of the OPEN bonds
by a factor exp(eps * N(0,1)) on the device, hands the list to pn_update_conductances and calls pn_solve again: no
host-to-device copy of the network, labelling and peeling reused while no bond crosses zero, warm start from the
previous pressures.  `--flip K` additionally closes K open bonds per step (a topology change: labels are redone).
One JSON line per step: seconds, inner iterations, labels_reused, G_eff.  Inputs are synthetic and seeded.
Needs a CUDA device (there is no CPU fallback).
"""
from __future__ import annotations

import argparse
import json
import time


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="cfg4", choices=["cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--n", type=int, default=0)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--fraction", type=float, default=0.01)
    ap.add_argument("--eps", type=float, default=0.05)
    ap.add_argument("--flip", type=int, default=0)
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--seed", type=int, default=11)
    args = ap.parse_args()

    import torch
    from . import build, inputs, pn
    build.build()
    gen = {"cfg2": inputs.cfg2_fbm_2d, "cfg3": inputs.cfg3_percolation_3d, "cfg4": inputs.cfg4_fbm_cut_3d,
           "cfg5": inputs.cfg5_stratified_3d}[args.workload]
    if args.n:
        net = gen(args.n, args.n) if args.workload == "cfg2" else gen(args.n, args.n, args.n)
    else:
        net = gen()
    dev = [torch.from_numpy(g).cuda() for g in (net.gx, net.gy, net.gz) if g is not None]
    h = pn.Network(net.nx, net.ny, net.nz)
    gen_t = torch.Generator(device="cuda").manual_seed(args.seed)

    def solve(step):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        info = h.solve(net.directions[0], args.tol, accept=(pn.PN_OK,))
        fl = h.flux()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        print(json.dumps({"step": step, "network": net.name, "t_s": dt, "inner_iters": info.inner_iters,
                          "outer_cycles": info.outer_cycles, "labels_reused": info.labels_reused,
                          "t_label_ms": info.t_label_ms, "t_solve_ms": info.t_solve_ms, "rel_residual": info.rel_residual,
                          "g_eff": fl[2], "n_solved": info.n_solved, "n_peeled": info.n_peeled}), flush=True)

    h.set_conductances(*dev)
    solve(0)
    for step in range(1, args.steps + 1):
        axis, node, value = [], [], []
        for a, g in enumerate(dev):
            flat = g.reshape(-1)
            idx = torch.nonzero(flat > 0).reshape(-1)
            pick = idx[torch.randperm(idx.numel(), generator=gen_t, device="cuda")[:max(1, int(args.fraction * idx.numel()))]]
            new = flat[pick] * torch.exp(args.eps * torch.randn(pick.numel(), generator=gen_t, device="cuda"))
            new = new.clamp_min(1e-6).to(torch.float32)
            if args.flip:
                new[:args.flip] = 0.0
            flat[pick] = new                      # the caller's own copy follows the network
            axis.append(torch.full((pick.numel(),), a, dtype=torch.int32, device="cuda"))
            node.append(pick.to(torch.int64))
            value.append(new)
        t0 = time.perf_counter()
        h.update_conductances(torch.cat(axis), torch.cat(node), torch.cat(value))
        torch.cuda.synchronize()
        t_upd = time.perf_counter() - t0
        solve(step)
        print(json.dumps({"step": step, "t_update_s": t_upd, "bonds_changed": int(sum(v.numel() for v in value))}), flush=True)
    h.close()


if __name__ == "__main__":
    main()
