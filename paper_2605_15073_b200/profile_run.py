"""Runs a few steps of one BASELINE.json config through the C ABI -- the small, fixed command that the
ncu captures under profiles/ are made with.

    python -m paper_2605_15073_b200.profile_run --config 1 --steps 2            # on-site, configs[1]
    python -m paper_2605_15073_b200.profile_run --config 3 --lmax 20 --steps 1  # on-site sweep point
    python -m paper_2605_15073_b200.profile_run --config 4 --steps 1            # message passing, configs[4]
    python -m paper_2605_15073_b200.profile_run --config 1 --math-mode 1        # 3xTF32 tensor-core projections
    python -m paper_2605_15073_b200.profile_run --config 1 --nu 3               # nu-body product at the shape of configs[1]
    python -m paper_2605_15073_b200.profile_run --config 2 --edge-field 128     # two-field coupling on the graph of configs[2]
    python -m paper_2605_15073_b200.profile_run --kernel-path 16 --config 1     # four-launch on-site step (CGTP_PATH_*)
    python -m paper_2605_15073_b200.profile_run --sanitize                      # one small call of every kernel family
                                                                                # (the compute-sanitizer command)
"""
from __future__ import annotations

import argparse

import numpy as np
import torch

from . import binding as cg
from . import synthetic


def sanitize():
    """One small call of every kernel family that uses mbarriers / TMA rings / named barriers, for compute-sanitizer
    (memcheck, racecheck): proj_fast, proj_multi, proj_tc, onsite_fused, onsite_fast (both parities, row-blocked form at
    band limit 12), onsite_generic, nbody_core, segments, node synthesis (fast and generic), edge_ring, edge_kernel,
    edge_lr, analysis, field gather / pool, sigma mask."""
    dev = torch.device("cuda", 0)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    n = 0

    def onsite(lmax, N, C, batch, path=0, mode=0):
        inp = synthetic.make_onsite(lmax, lmax, N, C, batch, seed=1)
        cg.cgtp_set_kernel_path(path)
        cg.cgtp_set_math_mode(mode)
        cg.cgtp_onsite(cu(inp.A), cu(inp.B), cu(inp.W_a), cu(inp.W_b), cu(inp.W_out), lmax, lmax, N, C, inp.parity_mask)
        cg.cgtp_set_kernel_path(0)
        cg.cgtp_set_math_mode(0)

    onsite(2, 8, 8, 64)                                  # configs[0]: onsite_fused (roomy layout)
    onsite(6, 64, 64, 20)                                # onsite_fused (tight layout)
    onsite(6, 64, 64, 70, path=cg.PATH_UNFUSED_ONSITE | cg.PATH_SMEM_CORE)  # proj_fast + onsite_fast
    onsite(4, 16, 16, 70, path=cg.PATH_UNFUSED_ONSITE)   # onsite_reg (one thread per column)
    onsite(12, 8, 8, 40, path=cg.PATH_UNFUSED_ONSITE)    # onsite_fast, row blocks
    onsite(4, 16, 16, 50, path=cg.PATH_UNFUSED_ONSITE | cg.PATH_GENERIC_CORE | cg.PATH_GENERIC_PROJ)
    onsite(4, 24, 40, 70, path=cg.PATH_UNFUSED_ONSITE, mode=cg.MATH_3XTF32)  # proj_tc (tcgen05)
    n += 6
    inp = synthetic.make_onsite(3, 3, 8, 8, 40, seed=2)
    (Wa, Wb), Wo = synthetic.lw_weights(3, 3, 8, 8, seed=2)
    cg.cgtp_onsite_lw(cu(inp.A), cu(inp.B), cu(Wa), cu(Wb), cu(Wo), 3, 3, 8, 8, inp.parity_mask)  # proj_multi
    q = synthetic.make_onsite_parity(3, 3, 8, 4, 30, seed=3)
    cg.cgtp_onsite_parity(cu(q.A), cu(q.B), cu(q.W_a), cu(q.W_b), cu(q.W_out), 3, 3, 8, 4)        # ACC projections, sigma mask
    nb = synthetic.make_nbody(3, 3, 3, 8, 8, 40, seed=4)
    cg.cgtp_onsite_nbody(cu(nb.X), cu(nb.W_in), cu(nb.W_out), 3, 3, 3, 8, 8)
    n += 3
    for lmax, path in ((4, 0), (6, 0), (6, cg.PATH_GENERIC_EDGE | cg.PATH_GENERIC_SYNTH)):
        m = synthetic.make_message(lmax, lmax, 8, 16, 40, np.random.default_rng(lmax).integers(0, 12, 40), seed=5)
        cg.cgtp_set_kernel_path(path)
        cg.cgtp_message(cu(m.node_feats), cu(m.edge_index), cu(m.edge_vec), cu(m.edge_radial), cu(m.W_node), cu(m.W_out),
                        lmax, lmax, m.N, m.C, m.parity_mask, check=True)
        cg.cgtp_set_kernel_path(0)
        n += 1
    m = synthetic.make_message(4, 4, 8, 8, 30, 6, seed=6)
    (Wn,), Wo = synthetic.lw_weights(4, 4, 8, 8, seed=6, n_in=1)
    rad = np.ascontiguousarray(np.repeat(m.edge_radial[:, :, None], 5, axis=2))
    cg.cgtp_message_lwr(cu(m.node_feats), cu(m.edge_index), cu(m.edge_vec), cu(rad), cu(Wn), cu(Wo), 4, 4, 8, 8,
                        m.parity_mask, check=True)                                                  # edge_lr
    XE, We = synthetic.make_edge_field(m, 4, seed=6)
    cg.cgtp_message_field(cu(m.node_feats), cu(m.edge_index), cu(XE), cu(We), cu(m.W_node), cu(m.W_out), 4, 4, 8, 4, 8,
                          m.parity_mask, check=True)                                                # gather + pool
    f = synthetic.make_field_parity(3, 3, 4, 4, 4, 20, 5, seed=7)
    cg.cgtp_message_field_parity(cu(f.node_feats), cu(f.edge_index), cu(f.edge_feats), cu(f.W_edge), cu(f.W_node),
                                 cu(f.W_out), 3, 3, 4, 4, 4, check=True)
    n += 3
    torch.cuda.synchronize()
    print(f"sanitize: {n} calls, {cg.cgtp_launch_count()} launches")


def main():
    import sys
    if "--sanitize" in sys.argv:
        return sanitize()
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--lmax", type=int, default=None)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--batch", type=int, default=None, help="override the batch / node count")
    ap.add_argument("--all-even", action="store_true")
    ap.add_argument("--math-mode", type=int, default=0, help="0 FP32 (default), 1 3xTF32, 2 TF32 projections")
    ap.add_argument("--kernel-path", type=int, default=0, help="CGTP_PATH_* bits (include/cgtp.h)")
    ap.add_argument("--nu", type=int, default=0, help="> 0: cgtp_onsite_nbody with this body order at the on-site "
                    "config's lmax, N, C, batch (all rank channels pointwise)")
    ap.add_argument("--edge-field", type=int, default=0, help="> 0: cgtp_message_field on the graph of a message "
                    "config with an edge feature field of this many channels (Ne)")
    args = ap.parse_args()
    dev = torch.device("cuda", 0)
    cg.cgtp_set_math_mode(args.math_mode)
    cg.cgtp_set_kernel_path(args.kernel_path)
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
