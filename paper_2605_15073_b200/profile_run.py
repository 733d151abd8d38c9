"""Runs a few steps of one BASELINE.json config through the C ABI -- the small, fixed command that the
ncu captures under profiles/ are made with.

    python -m paper_2605_15073_b200.profile_run --config 1 --steps 2            # on-site, configs[1]
    python -m paper_2605_15073_b200.profile_run --config 3 --lmax 20 --steps 1  # on-site sweep point
    python -m paper_2605_15073_b200.profile_run --config 4 --steps 1            # message passing, configs[4]
    python -m paper_2605_15073_b200.profile_run --config 1 --math-mode 1        # 3xTF32 tensor-core projections
    python -m paper_2605_15073_b200.profile_run --config 1 --nu 3               # nu-body product at the shape of configs[1]
    python -m paper_2605_15073_b200.profile_run --config 2 --edge-field 128     # two-field coupling on the graph of configs[2]
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import binding as cg
from . import synthetic


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--lmax", type=int, default=None)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--batch", type=int, default=None, help="override the batch / node count")
    ap.add_argument("--all-even", action="store_true")
    ap.add_argument("--math-mode", type=int, default=0, help="0 FP32 (default), 1 3xTF32, 2 TF32 projections")
    ap.add_argument("--nu", type=int, default=0, help="> 0: cgtp_onsite_nbody with this body order at the on-site "
                    "config's lmax, N, C, batch (all rank channels pointwise)")
    ap.add_argument("--edge-field", type=int, default=0, help="> 0: cgtp_message_field on the graph of a message "
                    "config with an edge feature field of this many channels (Ne)")
    args = ap.parse_args()
    dev = torch.device("cuda", 0)
    cg.cgtp_set_math_mode(args.math_mode)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    inp = synthetic.config(args.config, lmax=args.lmax)
    if args.all_even:
        inp.parity_mask = np.zeros_like(inp.parity_mask)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.nu > 0:
        b = args.batch or inp.batch
        nb = synthetic.make_nbody(args.nu, inp.lmax, inp.lmax_out, inp.N, inp.C, b, seed=0)
        X, Wi, Wo = cu(nb.X), cu(nb.W_in), cu(nb.W_out)
        fn = lambda: cg.cgtp_onsite_nbody(X, Wi, Wo, nb.nu, nb.lmax, nb.lmax_out, nb.N, nb.C)
        units, unit = b, "products"
    elif isinstance(inp, synthetic.OnsiteInputs):
        b = args.batch or inp.batch
        A, B = cu(inp.A[:b]), cu(inp.B[:b])
        Wa, Wb, Wo = cu(inp.W_a), cu(inp.W_b), cu(inp.W_out)
        fn = lambda: cg.cgtp_onsite(A, B, Wa, Wb, Wo, inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask)
        units, unit = b, "contractions"
    elif args.edge_field > 0:
        XE, W_edge = synthetic.make_edge_field(inp, args.edge_field, seed=0)
        X, ei, XEd, We = cu(inp.node_feats), cu(inp.edge_index), cu(XE), cu(W_edge)
        Wn, Wo = cu(inp.W_node), cu(inp.W_out)
        fn = lambda: cg.cgtp_message_field(X, ei, XEd, We, Wn, Wo, inp.lmax, inp.lmax_out, inp.N, args.edge_field, inp.C,
                                           inp.parity_mask)
        units, unit = inp.E, "edges"
    else:
        X, ei, ev, er = cu(inp.node_feats), cu(inp.edge_index), cu(inp.edge_vec), cu(inp.edge_radial)
        Wn, Wo = cu(inp.W_node), cu(inp.W_out)
        fn = lambda: cg.cgtp_message(X, ei, ev, er, Wn, Wo, inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask)
        units, unit = inp.E, "edges"
    fn()
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        fn()
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    print(f"config {args.config}: {ms:.4f} ms/step, {units / ms * 1e3:.4g} {unit}/s, "
          f"launches {cg.cgtp_launch_count()}")


if __name__ == "__main__":
    main()
