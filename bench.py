#!/usr/bin/env python
"""bench.py -- throughput of the B200 contracted Clebsch-Gordan hot path (contract: see README/DESIGN.md).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]

One "step" = one pass of the whole on-site hot path (S1..S5: projection, Legendre/Fourier synthesis,
product / surface-curl pairing, analysis, output projection) over one batch of BASELINE.json configs[1]
(lmax=6, N=C=64, 4096 atoms, 32 even + 32 odd rank channels).  Metric: on-site contractions/s
(one contraction = one atom's full pipeline).  For N>1 (torchrun) every rank processes its own batch
(weak scaling, no collective on the data path).

Prints ONE JSON line on rank 0.  Extra objects on the line (N=1 only): "sweep" (configs[3], on-site vs
lmax), "message" (configs[2] and configs[4], edges/s and HBM GB/s), "kernels" (per-kernel shares), "parity"
(parity-labelled inputs: cost of the full dispatch against one Category-alpha run), "l_dependent_weights", "nbody"
(nu-body pointwise products), "edge_field" (two feature fields, Eq.(28)).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SM_COUNT = 148
FMA_LANES_PER_SM = 128  # 4 SMSPs x 32 FP32 lanes (B200_PROFILING.md / B300_MICROARCH.md unit counts)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


# ------------------------------------------------------------------------------------------------
# algorithmic work (SURVEY.md 8(d) / DESIGN.md "Measurement"): fixed formulas, minimal grid, dense DFT
# ------------------------------------------------------------------------------------------------
def grid_shape(lmax, lmax_out):
    return (2 * lmax + lmax_out + 2) // 2, 2 * lmax + lmax_out + 1


def onsite_flops_per_atom(lmax, lmax_out, N, C, Ce, Co):
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    U, V = grid_shape(lmax, lmax_out)
    M, Mo = 2 * lmax + 1, 2 * lmax_out + 1
    k = {
        "proj_in": 4 * C * N * L2,
        "onsite_core_even": Ce * (4 * U * L2 + 4 * U * V * M + U * V + 2 * U * V * Mo + 2 * U * Lo2),
        "onsite_core_odd": Co * (8 * U * L2 + 8 * U * V * M + 3 * U * V + 2 * U * V * Mo + 2 * U * Lo2),
        "proj_out": 2 * N * C * Lo2,
    }
    k["onsite_fused"] = sum(k.values())  # the single-kernel step (onsite_fused.cu) does all four
    return k


def onsite_bytes_per_atom(lmax, lmax_out, N):
    return 4 * (2 * N * (lmax + 1) ** 2 + 2 * N * (lmax_out + 1) ** 2)


def message_bytes(lmax, lmax_out, N, C, Ce, Co, nodes, E):
    """Algorithmic HBM bytes of the implemented data flow: every edge gathers ONE value grid per rank
    channel of either parity (the odd channels pair it with both derivative fields of the edge and pool two grids per
    receiver).  Also returns the total of SURVEY.md 8(d)'s "gather sender grids" flow (two gathered derivative fields per
    odd channel), which this build no longer moves, for comparison."""
    U, V = grid_shape(lmax, lmax_out)
    UV = U * V
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    k = {
        "edge_even": E * (4 * Ce * UV + 4 * Ce + 12 + 16) + nodes * 4 * Ce * UV,
        "edge_odd": E * (4 * Co * UV + 4 * Co + 12 + 16) + nodes * 8 * Co * UV,
    }
    total = E * (4 * C * UV + 4 * C + 12 + 16) + nodes * (4 * N * L2 + 4 * C * UV + 8 * N * Lo2)
    total_paper_flow = (E * (4 * (Ce + 2 * Co) * UV + 4 * C + 12 + 16)
                        + nodes * (4 * N * L2 + 4 * (Ce + 2 * Co) * UV + 8 * N * Lo2))
    return k, total, total_paper_flow


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML in a background thread."""

    def __init__(self, index: int, period: float = 0.02):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._t = None
        self.ok = False

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            return self
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8)),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40)),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20)),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)),
        }
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or getattr(
            nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(get_reasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop.set()
        if self._t:
            self._t.join()
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------
# reference arm = the oracle on the host cores
# ------------------------------------------------------------------------------------------------
def oracle_onsite_rate(inp, n_atoms, min_wall_s=0.0):
    """The oracle as it stands on the host cores: passes over the first n_atoms atoms until min_wall_s of wall time has
    gone by (at least one pass).  Returns (atoms/s, wall seconds, threads, passes)."""
    from oracle import cgtp_oracle as orc
    n = min(n_atoms, inp.batch)
    orc.real_coupling(inp.lmax, inp.lmax_out, False)
    orc.real_coupling(inp.lmax, inp.lmax_out, True)  # tables are set-up, not the timed work
    t0 = time.perf_counter()
    passes = 0
    while True:
        orc.onsite(inp.A[:n], inp.B[:n], inp.W_a, inp.W_b, inp.W_out, inp.lmax, inp.lmax_out, inp.parity_mask)
        passes += 1
        dt = time.perf_counter() - t0
        if dt >= min_wall_s:
            break
    return n * passes / dt, dt, orc.num_threads(), passes


def run_reference(args, rank, world):
    if rank != 0:
        return
    from paper_2605_15073_b200 import synthetic
    inp = synthetic.config(1)
    n = 1024
    from oracle import cgtp_oracle as orc
    orc.real_coupling(inp.lmax, inp.lmax_out, False)
    orc.real_coupling(inp.lmax, inp.lmax_out, True)
    for _ in range(max(args.warmup, 1)):
        oracle_onsite_rate(inp, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_onsite_rate(inp, n)
    dt = time.perf_counter() - t0
    val = n * args.steps / dt
    line = {
        "impl": "reference", "metric": "onsite_contractions_per_s", "value": val, "unit": "contractions/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: on-site lmax=6 lmax_out=6 N=64 C=64 batch=4096 even+odd",
                   "sample": f"first {n} atoms per step"},
        "cpu_baseline": {"value": val, "unit": "contractions/s", "cores": orc.num_threads(), "kind": "oracle",
                         "sample": f"{n} of 4096 atoms per step, {args.steps} steps"},
        "e2e": {"value": val, "unit": "contractions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--sweep-batch", type=int, default=16384)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    from paper_2605_15073_b200 import binding as cg
    from paper_2605_15073_b200 import synthetic

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cg.lib()  # fails loudly if the CUDA library is missing

    peaks, peak_src = load_peaks()
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ------------------------------------------------------------------ main workload: configs[1]
    NSETS = 4  # rotating input sets: 4 x (A,B) = 411 MB > 126 MB L2, so no step finds its inputs in L2
    sets = []
    base = None
    for s in range(NSETS):
        inp = synthetic.config(1, seed=1000 * rank + s)
        base = base or inp
        sets.append((cu(inp.A), cu(inp.B)))
    Wa, Wb, Wo = cu(base.W_a), cu(base.W_b), cu(base.W_out)
    lmax, lmax_out, N, C, batch, mask = base.lmax, base.lmax_out, base.N, base.C, base.batch, base.parity_mask
    Ce, Co = int((mask == 0).sum()), int((mask == 1).sum())
    out = torch.empty((batch, 2, N, (lmax_out + 1) ** 2), dtype=torch.float32, device=dev)

    def step(i):
        A, B = sets[i % NSETS]
        cg.cgtp_onsite(A, B, Wa, Wb, Wo, lmax, lmax_out, N, C, mask, out=out)

    # FP32 pipe calibration in the same run: register-only FFMA / FFMA2 chains on every SM
    ffma_tf, ffma_mhz = cg.cgtp_fma_peak(False, 30.0)
    ffma2_tf, ffma2_mhz = cg.cgtp_fma_peak(True, 30.0)
    fp32_peak_measured = max(ffma_tf, ffma2_tf)

    sampler = ClockSampler(local_rank).start()
    for i in range(args.warmup):
        step(i)
    barrier()
    l0 = cg.cgtp_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for i in range(args.steps):
        step(i)
    ev1.record()
    barrier()
    ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    launches = cg.cgtp_launch_count() - l0
    ms_per_step = ms_total / args.steps
    value = world * batch / (ms_per_step * 1e-3)

    # keep the same load running so that the clock record covers >= ~1 s of it
    t_end = time.perf_counter() + 1.0
    i = 0
    while time.perf_counter() < t_end:
        for _ in range(20):
            step(i)
            i += 1
        torch.cuda.synchronize()
    clocks = sampler.stop()

    # per-kernel durations over another K steps (CUDA events around every launch, on the launch stream)
    cg.cgtp_profile_enable(True)
    for i in range(args.steps):
        step(i)
    torch.cuda.synchronize()
    prof = cg.cgtp_profile_collect()
    cg.cgtp_profile_enable(False)

    fl = onsite_flops_per_atom(lmax, lmax_out, N, C, Ce, Co)
    step_flops = fl["proj_in"] + fl["onsite_core_even"] + fl["onsite_core_odd"] + fl["proj_out"]
    sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz", 1965.0)
    fp32_peak_tflops = SM_COUNT * FMA_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    kernels = {}
    for name, (ms, cnt) in prof.items():
        avg_ms = ms / cnt
        k = {"launches_per_step": cnt / args.steps, "avg_ms": avg_ms}
        if name in fl:
            k["alg_tflops"] = fl[name] * batch / (avg_ms * 1e-3) / 1e12
            k["frac_fp32_peak"] = k["alg_tflops"] / fp32_peak_tflops
        kernels[name] = k
    tot_ms = sum(ms for ms, _ in prof.values())
    for name, (ms, cnt) in prof.items():
        kernels[name]["share"] = ms / tot_ms
    dom = max(prof, key=lambda n: prof[n][0])
    traffic = pipe_util = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        tj = json.load(open(tp))
        traffic = tj.get(f"config1:{dom}")
        pipe_util = tj.get(f"config1:{dom}:pipe_util")
    roofline = {
        "kernel": dom, "bound": "alu", "achieved": kernels[dom]["alg_tflops"], "peak": fp32_peak_tflops,
        "unit": "TFLOP/s", "frac": kernels[dom]["alg_tflops"] / fp32_peak_tflops, "traffic": traffic,
        "peak_source": f"derived: {SM_COUNT} SMs x {FMA_LANES_PER_SM} FP32 FMA lanes x 2 x {sm_max:.0f} MHz (DESIGN.md)",
        "peak_measured": fp32_peak_measured,
        "peak_measured_source": "cgtp_fma_peak in this run: register-only dependent chains on every SM, 30 ms each: "
                                f"FFMA {ffma_tf:.1f} TFLOP/s (= {ffma_mhz:.0f} MHz x 148 x 128 x 2), FFMA2 {ffma2_tf:.1f} TFLOP/s",
        "frac_of_measured": kernels[dom]["alg_tflops"] / fp32_peak_measured,
        "pipe_util": pipe_util,
        "pipe_util_definition": "ncu counters of the kept capture of this kernel (file named inside): FMA-pipe cycles "
                                "active, issue slots used, shared-memory wavefronts -- `frac` counts the paper's dense "
                                "transforms, the kernel folds symmetries, so frac > pipe utilisation is expected",
        "achieved_definition": "algorithmic FP32 flops of this kernel per launch (SURVEY.md 8(d) formula, dense DFT, "
                               "no symmetry folding) / mean CUDA-event duration",
        "step_alg_tflops": step_flops * batch / (ms_per_step * 1e-3) / 1e12,
        "step_frac_fp32_peak": step_flops * batch / (ms_per_step * 1e-3) / 1e12 / fp32_peak_tflops,
        "step_frac_of_measured": step_flops * batch / (ms_per_step * 1e-3) / 1e12 / fp32_peak_measured,
        "step_hbm_gbs_algorithmic": onsite_bytes_per_atom(lmax, lmax_out, N) * batch / (ms_per_step * 1e-3) / 1e9,
        "hbm_peak_gbs": peaks["hbm_gbs"], "hbm_peak_source": peak_src,
    }

    # ------------------------------------------------------------------ end to end with host buffers
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hA, hB = pin(base.A), pin(base.B)
    hWa, hWb, hWo = pin(base.W_a), pin(base.W_b), pin(base.W_out)
    hout = torch.empty((batch, 2, N, (lmax_out + 1) ** 2), dtype=torch.float32).pin_memory()
    ke = max(3, min(args.steps, 20))
    for _ in range(2):
        cg.cgtp_onsite_host(hA, hB, hWa, hWb, hWo, lmax, lmax_out, N, C, mask, out=hout)
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        cg.cgtp_onsite_host(hA, hB, hWa, hWb, hWo, lmax, lmax_out, N, C, mask, out=hout)
    torch.cuda.synchronize()
    dt = max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * batch * ke / dt, "unit": "contractions/s",
           "h2d_bytes_per_step": int(hA.numel() + hB.numel() + hWa.numel() + hWb.numel() + hWo.numel()) * 4,
           "d2h_bytes_per_step": int(hout.numel()) * 4, "steps": ke, "ms_per_step": 1e3 * dt / ke}

    line = {
        "metric": "onsite_contractions_per_s", "value": value, "unit": "contractions/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: on-site lmax=6 lmax_out=6 N=64 C=64 batch=4096/GPU, "
                               "32 even + 32 odd rank channels",
                   "l2": f"{NSETS} rotating input sets (411 MB) + 360 MB touched per step > 126 MB L2",
                   "parallelism": f"dp{world} (batch split, no collective)"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "kernels": kernels,
    }

    # ------------------------------------------------------------------ receiver-sharded message passing (every N)
    if not args.no_extras:
        line["message_sharded"] = run_message_sharded(args, cg, synthetic, dev, rank, world, peaks, barrier, max_over_ranks)

    # ------------------------------------------------------------------ extras (rank 0, 1 GPU)
    if world == 1 and not args.no_extras:
        sampler2 = ClockSampler(local_rank, period=0.05).start()  # the extras get their own clock record
        rate, dt_cpu, cores, passes = oracle_onsite_rate(base, batch, min_wall_s=1.5)
        line["cpu_baseline"] = {"value": rate, "unit": "contractions/s", "cores": cores, "kind": "oracle",
                                "sample": f"all {batch} atoms of configs[1], {passes} passes ({dt_cpu:.1f} s wall, "
                                          f"{dt_cpu * cores:.0f} s of CPU work)"}
        line["tensor_core"] = run_tensor_core(args, cg, step, out, lmax, lmax_out, N, C, Ce, Co, batch, peaks, peak_src)
        line["sweep"] = run_sweep(args, cg, synthetic, dev, fp32_peak_tflops, peaks)
        line["message"] = run_message(args, cg, synthetic, dev, peaks, peak_src)
        line["parity"] = run_parity(args, cg, synthetic, dev)
        line["l_dependent_weights"] = run_lw(args, cg, synthetic, dev, ms_per_step)
        line["nbody"] = run_nbody(args, cg, synthetic, dev, fp32_peak_tflops)
        line["edge_field"] = run_edge_field(args, cg, synthetic, dev, fp32_peak_tflops)
        # the other on-site path beside the library's own choice (four launches at configs[1] since the projections address
        # with compile-time strides): the single fused kernel, forced
        line["fused_onsite"] = run_other_path(args, cg, step, fl, batch, fp32_peak_tflops, fp32_peak_measured,
                                              cg.PATH_FUSED_ONSITE)
        line["clocks_extras"] = sampler2.stop()
    elif world == 1:
        rate, dt_cpu, cores, passes = oracle_onsite_rate(base, 1024, min_wall_s=1.0)
        line["cpu_baseline"] = {"value": rate, "unit": "contractions/s", "cores": cores, "kind": "oracle",
                                "sample": f"first 1024 atoms of configs[1], {passes} passes ({dt_cpu:.1f} s wall)"}

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def time_steps(fn, steps, warmup):
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(steps):
        fn()
    ev1.record()
    torch.cuda.synchronize()
    return ev0.elapsed_time(ev1) / steps


def run_message_sharded(args, cg, synthetic, dev, rank, world, peaks, barrier, max_over_ranks):
    """BASELINE.json configs[4] split over the ranks by receivers: every rank owns a
    contiguous receiver range, its in-edges and its rows of node_feats; one all-gather of node_feats (NCCL), then
    cgtp_message_bipartite over the local in-edges.  Strong scaling: the graph is fixed, edges/s = E / max-over-ranks
    time of (all-gather + kernels).  At N = 1 the all-gather is the identity and the call is cgtp_message itself."""
    import torch
    import torch.distributed as dist
    from paper_2605_15073_b200 import parallel
    m = synthetic.config(4)
    rp = parallel.row_ptr_from_receivers(m.edge_index[1], m.nodes)
    bounds = parallel.shard_receivers(rp, world)
    t = torch.from_numpy
    sh = parallel.make_shard(t(m.node_feats), t(m.edge_index), t(m.edge_vec), t(m.edge_radial), bounds, rank, row_ptr=rp)
    local = sh.node_feats.to(dev)
    ei, ev, er = sh.edge_index.to(dev), sh.edge_vec.to(dev), sh.edge_radial.to(dev)
    Wn, Wo = t(m.W_node).to(dev), t(m.W_out).to(dev)
    feats = torch.empty((m.nodes, m.N, (m.lmax + 1) ** 2), device=dev)
    out = torch.empty((sh.hi - sh.lo, 2, m.N, (m.lmax_out + 1) ** 2), device=dev)
    steps = max(3, min(args.steps, 10))
    ev_a0, ev_a1, ev_k1 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    ag_ms, tot_ms = [], []

    def one(timed):
        ev_a0.record()
        full = parallel.all_gather_node_feats(local, bounds, out=feats) if world > 1 else local
        ev_a1.record()
        cg.cgtp_message_bipartite(full, ei, ev, er, Wn, Wo, m.lmax, m.lmax_out, m.N, m.C, m.parity_mask, sh.hi - sh.lo, out=out)
        ev_k1.record()
        if timed:
            torch.cuda.synchronize()
            ag_ms.append(ev_a0.elapsed_time(ev_a1))
            tot_ms.append(ev_a0.elapsed_time(ev_k1))
    for _ in range(3):
        one(False)
    for _ in range(steps):
        barrier()
        one(True)
    step_ms = max_over_ranks(float(np.mean(tot_ms)))
    gather_ms = max_over_ranks(float(np.mean(ag_ms)))
    gathered_bytes = feats.numel() * 4 * (world - 1) / max(world, 1)  # bytes every rank receives
    return {"workload": f"BASELINE.json configs[4] over {world} receiver shard(s): nodes={m.nodes} E={m.E}, rank 0 owns "
                        f"receivers [{int(bounds[0])}, {int(bounds[1])}) with {int(ei.shape[1])} in-edges",
            "scaling": "strong", "ranks": world,
            "backend": dist.get_backend() if world > 1 else "none (single process)",
            "ms_per_step": step_ms, "edges_per_s": m.E / (step_ms * 1e-3),
            "all_gather_ms": gather_ms,
            "all_gather_gbs_per_rank": (gathered_bytes / (gather_ms * 1e-3) / 1e9) if world > 1 and gather_ms > 0 else None,
            "all_gather_bytes_per_rank": int(gathered_bytes), "steps": steps,
            "timing": "CUDA events on the launch stream around all-gather + kernels, mean over steps, max over ranks"}


def run_other_path(args, cg, step, fl, batch, fp32_peak_tflops, fp32_peak_measured, path):
    """configs[1] through the on-site path the library did NOT choose, forced with a CGTP_PATH_* flag
    (CGTP_PATH_FUSED_ONSITE: S1-S5 in one kernel, onsite_fused.cu; CGTP_PATH_UNFUSED_ONSITE: proj_fast + core x 2 +
    proj_fast): what the headline step is measured against."""
    import torch
    try:
        cg.cgtp_set_kernel_path(path)
        it = [0]

        def fn():
            it[0] += 1
            step(it[0])
        ms = time_steps(fn, max(args.steps // 2, 5), 3)
        cg.cgtp_profile_enable(True)
        for _ in range(20):
            fn()
        torch.cuda.synchronize()
        prof = cg.cgtp_profile_collect()
        cg.cgtp_profile_enable(False)
    finally:
        cg.cgtp_set_kernel_path(0)
    kern = {}
    for k, (kms, cnt) in prof.items():
        a = kms / cnt
        kern[k] = {"avg_ms": a}
        if k in fl:
            kern[k]["alg_tflops"] = fl[k] * batch / (a * 1e-3) / 1e12
            kern[k]["frac_fp32_peak"] = kern[k]["alg_tflops"] / fp32_peak_tflops
            kern[k]["frac_of_measured"] = kern[k]["alg_tflops"] / fp32_peak_measured
    return {"kernel_path": int(path), "ms_per_step": ms, "contractions_per_s": batch / (ms * 1e-3), "kernels": kern}


def run_tensor_core(args, cg, step, out, lmax, lmax_out, N, C, Ce, Co, batch, peaks, peak_src):
    """configs[1] with the channel projections (S1, S5) on tcgen05 tensor cores: 3xTF32 and single-pass TF32
    (cgtp_set_math_mode).  Reported beside, never inside, the FP32 headline `value`."""
    import torch
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    fl = onsite_flops_per_atom(lmax, lmax_out, N, C, Ce, Co)
    # compulsory bytes of the projection kernels: read X once, write the product once
    by = {"proj_in": 4 * (2 * N * L2 + 2 * C * L2) * batch, "proj_out": 4 * (C * Lo2 + 2 * N * Lo2) * batch}
    tf32_peak = peaks["bf16_tflops"] * 0.5  # nominal TF32 : bf16 ratio (B200_PROFILING.md table)
    step(0)
    torch.cuda.synchronize()
    ref = out.clone()
    res = {"tf32_peak_tflops": tf32_peak, "tf32_peak_source": f"{peak_src} bf16 peak x 0.5 (nominal TF32:bf16)"}
    try:
        for name, mode, passes in (("3xtf32", cg.MATH_3XTF32, 3), ("tf32", cg.MATH_TF32, 1)):
            cg.cgtp_set_math_mode(mode)
            ms = time_steps(lambda: step(0), max(args.steps // 2, 5), 3)
            err = [float((out[:, s] - ref[:, s]).abs().max() / ref[:, s].abs().max()) for s in (0, 1)]
            cg.cgtp_profile_enable(True)
            for i in range(20):
                step(i)
            torch.cuda.synchronize()
            prof = cg.cgtp_profile_collect()
            cg.cgtp_profile_enable(False)
            kern = {}
            for k in ("proj_in", "proj_out"):
                kms = prof[k][0] / prof[k][1]
                kern[k] = {"avg_ms": kms, "alg_hbm_gbs": by[k] / (kms * 1e-3) / 1e9,
                           "frac_hbm_peak": by[k] / (kms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                           "mma_tflops": passes * fl[k] * batch / (kms * 1e-3) / 1e12,
                           "frac_tf32_peak": passes * fl[k] * batch / (kms * 1e-3) / 1e12 / tf32_peak}
            res[name] = {"ms_per_step": ms, "contractions_per_s": batch / (ms * 1e-3),
                         "max_rel_diff_vs_fp32_path": err, "bound": "hbm", "kernels": kern}
    finally:
        cg.cgtp_set_math_mode(cg.MATH_FP32)
    return res


def run_sweep(args, cg, synthetic, dev, fp32_peak_tflops, peaks):
    """BASELINE.json configs[3]: on-site, N=C=32, batch=16384, lmax in {2,4,8,12,16,20} (inputs drawn on the
    device with a seeded torch generator: same distribution as synthetic.make_onsite)."""
    import torch
    res = []
    N = C = 32
    batch = args.sweep_batch
    g = torch.Generator(device=dev)
    g.manual_seed(3)
    mask = synthetic.half_mask(C)
    Wa = torch.randn((C, N), generator=g, device=dev) / N ** 0.5
    Wb = torch.randn((C, N), generator=g, device=dev) / N ** 0.5
    Wo = torch.randn((N, C), generator=g, device=dev) / C ** 0.5
    for lmax in (2, 4, 8, 12, 16, 20):
        L2 = (lmax + 1) ** 2
        A = torch.randn((batch, N, L2), generator=g, device=dev)
        B = torch.randn((batch, N, L2), generator=g, device=dev)
        out = torch.empty((batch, 2, N, L2), device=dev)
        fn = lambda: cg.cgtp_onsite(A, B, Wa, Wb, Wo, lmax, lmax, N, C, mask, out=out)
        steps = 20 if lmax <= 8 else 5
        ms = time_steps(fn, steps, 3)
        cg.cgtp_profile_enable(True)
        for _ in range(steps):
            fn()
        torch.cuda.synchronize()
        prof = cg.cgtp_profile_collect()
        cg.cgtp_profile_enable(False)
        fls = onsite_flops_per_atom(lmax, lmax, N, C, C // 2, C // 2)
        fl = fls["onsite_fused"]
        by = onsite_bytes_per_atom(lmax, lmax, N)
        res.append({"lmax": lmax, "ms_per_step": ms, "contractions_per_s": batch / (ms * 1e-3),
                    "kernel_ms": {k: v[0] / v[1] * (v[1] / steps) for k, v in prof.items()},
                    "alg_tflops": fl * batch / (ms * 1e-3) / 1e12,
                    "frac_fp32_peak": fl * batch / (ms * 1e-3) / 1e12 / fp32_peak_tflops,
                    "alg_hbm_gbs": by * batch / (ms * 1e-3) / 1e9,
                    "frac_hbm_peak": by * batch / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"]})
        del A, B, out
    return {"workload": f"BASELINE.json configs[3]: on-site N=C=32 batch={batch} lmax_out=lmax, 16 even + 16 odd",
            "points": res}


def run_message(args, cg, synthetic, dev, peaks, peak_src):
    import torch
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    res = {}
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    ncu_traffic = json.load(open(tp)) if os.path.exists(tp) else {}
    for name, idx, halfhalf in (("config2_all_even", 2, False), ("config2_half_odd", 2, True), ("config4", 4, True)):
        m = synthetic.config(idx)
        if idx == 2 and halfhalf:
            m.parity_mask = synthetic.half_mask(m.C)
        Ce, Co = int((m.parity_mask == 0).sum()), int((m.parity_mask == 1).sum())
        X, ei, ev, er = cu(m.node_feats), cu(m.edge_index), cu(m.edge_vec), cu(m.edge_radial)
        Wn, Wo = cu(m.W_node), cu(m.W_out)
        out = torch.empty((m.nodes, 2, m.N, (m.lmax_out + 1) ** 2), device=dev)
        fn = lambda: cg.cgtp_message(X, ei, ev, er, Wn, Wo, m.lmax, m.lmax_out, m.N, m.C, m.parity_mask, out=out)
        steps = max(3, min(args.steps, 50 if idx == 2 else 10))
        ms = time_steps(fn, steps, 3)
        cg.cgtp_profile_enable(True)
        for _ in range(steps):
            fn()
        torch.cuda.synchronize()
        prof = cg.cgtp_profile_collect()
        cg.cgtp_profile_enable(False)
        kb, total_bytes, paper_bytes = message_bytes(m.lmax, m.lmax_out, m.N, m.C, Ce, Co, m.nodes, m.E)
        kern = {}
        tot = sum(v[0] for v in prof.values())
        for k, (kms, cnt) in prof.items():
            kern[k] = {"avg_ms": kms / cnt, "share": kms / tot}
            if k in kb:
                kern[k]["alg_gbs"] = kb[k] / (kms / cnt * 1e-3) / 1e9
                kern[k]["frac_hbm_peak"] = kern[k]["alg_gbs"] / peaks["hbm_gbs"]
        dom = max(prof, key=lambda n: prof[n][0])
        res[name] = {
            "workload": f"BASELINE.json configs[{idx}]: nodes={m.nodes} E={m.E} lmax={m.lmax} N=C={m.C} "
                        f"even={Ce} odd={Co}",
            "ms_per_step": ms, "edges_per_s": m.E / (ms * 1e-3),
            "alg_hbm_gbs_whole_step": total_bytes / (ms * 1e-3) / 1e9,
            "frac_hbm_peak_whole_step": total_bytes / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "paper_flow_equiv_gbs": paper_bytes / (ms * 1e-3) / 1e9,
            "numerator": "implemented flow: one gathered value grid per (edge, channel); paper_flow_equiv_gbs uses "
                         "SURVEY.md 8(d)'s two-derivative-field gather for the odd channels",
            "roofline": {"kernel": dom, "bound": "hbm", "achieved": kern[dom].get("alg_gbs"),
                         "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": kern[dom].get("frac_hbm_peak"),
                         "peak_source": peak_src, "traffic": ncu_traffic.get(f"config{idx}:{dom}") if halfhalf else None},
            "kernels": kern,
        }
        if idx == 4:
            # M1 / M6 on the tensor cores (tcgen05, 3xTF32: three TF32 products per FP32 product), reported beside the
            # FP32-exact step, never inside it (north_star: "TF32/3xTF32 reported separately")
            ref_out = out.clone()
            cg.cgtp_set_math_mode(cg.MATH_3XTF32)
            try:
                ms_tc = time_steps(fn, steps, 3)
                fn()
                torch.cuda.synchronize()
                diff = [float((out[:, s_] - ref_out[:, s_]).abs().max() / ref_out[:, s_].abs().max()) for s_ in (0, 1)]
            finally:
                cg.cgtp_set_math_mode(cg.MATH_FP32)
            res[name]["projections_3xtf32"] = {
                "ms_per_step": ms_tc, "edges_per_s": m.E / (ms_tc * 1e-3),
                "frac_hbm_peak_whole_step": total_bytes / (ms_tc * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "max_rel_diff_vs_fp32_path": diff}
            del ref_out
        if idx == 2:
            # the node-grid table the edges gather from (95 MB) is written by M2 in the same step and stays in the 126 MB
            # L2 (SURVEY.md 8(d) says so): the gather is an L2 read, the algorithmic rate is not an HBM measurement
            r = res[name]["roofline"]
            r.update({"bound": "l2", "peak": None, "frac": None, "peak_source": None,
                      "note": "gathered table is L2-resident; `achieved` = algorithmic gather bytes / time; the ncu "
                              "capture (lts__t_bytes, dram__bytes) is in profiles/, see traffic.json",
                      "traffic": ncu_traffic.get(f"config2:{dom}"), "l2_bytes": ncu_traffic.get(f"config2:{dom}:lts_bytes")})
            for kk in kern.values():
                kk.pop("frac_hbm_peak", None)
            res[name].pop("frac_hbm_peak_whole_step", None)
        del X, ei, ev, er, out
        torch.cuda.empty_cache()
    return res


def run_parity(args, cg, synthetic, dev):
    """Parity-labelled inputs (Sec. VII C a-c, e): cost of the full (p, sigma) dispatch
    relative to ONE Category-alpha run of the same N and C -- the unit of the paper's 12x (Eq.(60) :455) and 24x (:469)
    upper bounds.  Shapes: configs[1] / configs[2] with C/4 rank channels per run, so a pass has the configs' C."""
    import torch
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    res = {}
    # on-site: lmax=6, N=64, C=16 per run (16 runs, 4 passes of 64 internal channels), 4096 atoms
    q = synthetic.make_onsite_parity(6, 6, 64, 16, 4096, seed=0)
    A, B, Wa, Wb, Wo = cu(q.A), cu(q.B), cu(q.W_a), cu(q.W_b), cu(q.W_out)
    out = torch.empty((q.batch, 2, q.N, 49), device=dev)
    ms = time_steps(lambda: cg.cgtp_onsite_parity(A, B, Wa, Wb, Wo, 6, 6, q.N, q.C, out=out), 20, 3)
    A0, B0 = A[:, 0].contiguous(), B[:, 0].contiguous()
    Wa0, Wb0, Wo0 = Wa[0].contiguous(), Wb[0].contiguous(), Wo[0].contiguous()
    mask0 = np.zeros(q.C, np.uint8)
    ms1 = time_steps(lambda: cg.cgtp_onsite(A0, B0, Wa0, Wb0, Wo0, 6, 6, q.N, q.C, mask0, out=out), 20, 3)
    res["onsite"] = {"workload": "lmax=6 N=64 C=16 per run x 16 runs, batch=4096, both slots populated",
                     "ms_per_step": ms, "contractions_per_s": q.batch / (ms * 1e-3), "alpha_run_ms": ms1,
                     "factor_vs_alpha_run": ms / ms1, "paper_upper_bound": 24}
    del A, B, out, A0, B0
    # message passing: configs[2] graph, lmax=4, N=128, C=32 per run (8 runs, 2 passes of 128 internal channels)
    m = synthetic.make_message_parity(4, 4, 128, 32, 2048, 16, 0.8, 5.0, seed=0)
    X, ei, ev, er, Wn, Wo = cu(m.node_feats), cu(m.edge_index), cu(m.edge_vec), cu(m.edge_radial), cu(m.W_node), cu(m.W_out)
    out = torch.empty((m.nodes, 2, m.N, 25), device=dev)
    ms = time_steps(lambda: cg.cgtp_message_parity(X, ei, ev, er, Wn, Wo, 4, 4, m.N, m.C, out=out), 10, 3)
    X0, er0, Wn0, Wo0 = X[:, 0].contiguous(), er[:, 0].contiguous(), Wn[0].contiguous(), Wo[0].contiguous()
    mask0 = np.zeros(m.C, np.uint8)
    ms1 = time_steps(lambda: cg.cgtp_message(X0, ei, ev, er0, Wn0, Wo0, 4, 4, m.N, m.C, mask0, out=out), 10, 3)
    res["message"] = {"workload": "configs[2] graph (2048 nodes, 32768 edges), lmax=4 N=128 C=32 per run x 8 runs",
                      "ms_per_step": ms, "edges_per_s": m.E / (ms * 1e-3), "alpha_run_ms": ms1,
                      "factor_vs_alpha_run": ms / ms1, "paper_upper_bound": 12}
    del X, ei, ev, er, out
    # two parity-bearing fields (Eq.(28) :236, Sec. VII C f :471): configs[2] graph, lmax=4, N=128, Ne=8, C=32 per run x 16 runs
    f = synthetic.make_field_parity(4, 4, 128, 8, 32, 2048, 16, seed=0)
    X, ei, XE = cu(f.node_feats), cu(f.edge_index), cu(f.edge_feats)
    We, Wn, Wo = cu(f.W_edge), cu(f.W_node), cu(f.W_out)
    out = torch.empty((f.nodes, 2, f.N, 25), device=dev)
    ms = time_steps(lambda: cg.cgtp_message_field_parity(X, ei, XE, We, Wn, Wo, 4, 4, f.N, f.Ne, f.C, out=out), 10, 3)
    X0, XE0 = X[:, 0].contiguous(), XE[:, 0].contiguous()
    We0, Wn0, Wo0 = We[0].contiguous(), Wn[0].contiguous(), Wo[0].contiguous()
    mask0 = np.zeros(f.C, np.uint8)
    ms1 = time_steps(lambda: cg.cgtp_message_field(X0, ei, XE0, We0, Wn0, Wo0, 4, 4, f.N, f.Ne, f.C, mask0, out=out), 10, 3)
    res["field"] = {"workload": "configs[2] graph, edge field [E, 2, 8, 25], lmax=4 N=128 C=32 per run x 16 runs, both slots "
                                "of both fields populated",
                    "ms_per_step": ms, "edges_per_s": f.E / (ms * 1e-3), "alpha_run_ms": ms1,
                    "factor_vs_alpha_run": ms / ms1, "paper_upper_bound": 24}
    return res


def run_lw(args, cg, synthetic, dev, shared_ms):
    """l-dependent CP weights (Eq.(35), Eq.(41) :346): configs[1] with one weight
    matrix per degree; the channel projections run once per degree."""
    import torch
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    inp = synthetic.config(1)
    (Wa, Wb), Wo = synthetic.lw_weights(inp.lmax, inp.lmax_out, inp.N, inp.C, seed=0)
    A, B, Wa, Wb, Wo = cu(inp.A), cu(inp.B), cu(Wa), cu(Wb), cu(Wo)
    out = torch.empty((inp.batch, 2, inp.N, (inp.lmax_out + 1) ** 2), device=dev)
    fn = lambda: cg.cgtp_onsite_lw(A, B, Wa, Wb, Wo, inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask, out=out)
    ms = time_steps(fn, 20, 3)
    cg.cgtp_profile_enable(True)
    for _ in range(10):
        fn()
    torch.cuda.synchronize()
    prof = cg.cgtp_profile_collect()
    cg.cgtp_profile_enable(False)
    res_msg = {}
    for idx in (2, 4):
        m = synthetic.config(idx)
        if idx == 2:
            m.parity_mask = synthetic.half_mask(m.C)
        (Wn,), Wom = synthetic.lw_weights(m.lmax, m.lmax_out, m.N, m.C, seed=0, n_in=1)
        X, ei, ev, er = cu(m.node_feats), cu(m.edge_index), cu(m.edge_vec), cu(m.edge_radial)
        Wn, Wom = cu(Wn), cu(Wom)
        # R~[e, c, l1]: the configs' Bessel x Gaussian radial factor with a smooth l1 profile
        rad = (er[:, :, None] * torch.linspace(0.5, 1.5, m.lmax + 1, device=dev)[None, None, :]).contiguous()
        outm = torch.empty((m.nodes, 2, m.N, (m.lmax_out + 1) ** 2), device=dev)
        f_lw = lambda: cg.cgtp_message_lw(X, ei, ev, er, Wn, Wom, m.lmax, m.lmax_out, m.N, m.C, m.parity_mask, out=outm)
        f_lwr = lambda: cg.cgtp_message_lwr(X, ei, ev, rad, Wn, Wom, m.lmax, m.lmax_out, m.N, m.C, m.parity_mask, out=outm)
        ms_lw, ms_lwr = time_steps(f_lw, 3, 2), time_steps(f_lwr, 3, 2)
        res_msg[f"config{idx}"] = {
            "workload": f"BASELINE.json configs[{idx}] (half odd) with W_node [L, C, N], W_out [L, N, C]; lwr: edge_radial [E, C, L]",
            "lw_ms_per_step": ms_lw, "lw_edges_per_s": m.E / (ms_lw * 1e-3),
            "lwr_ms_per_step": ms_lwr, "lwr_edges_per_s": m.E / (ms_lwr * 1e-3)}
        del X, ei, ev, er, rad, outm
        torch.cuda.empty_cache()
    return {"message": res_msg,
            "workload": "BASELINE.json configs[1] with W_a, W_b [7, 64, 64] and W_out [7, 64, 64] (one matrix per degree)",
            "ms_per_step": ms, "contractions_per_s": inp.batch / (ms * 1e-3), "l_shared_ms_per_step": shared_ms,
            "factor_vs_l_shared": ms / shared_ms,
            "kernel_ms": {k: v[0] / 10 for k, v in prof.items()},
            "launches_per_step": int(sum(v[1] for v in prof.values()) // 10)}


def run_nbody(args, cg, synthetic, dev, fp32_peak_tflops):
    """nu-body pointwise products at the shape of configs[1] (all 64 rank channels
    pointwise) and at an ACE-like small band limit.  Algorithmic flops per atom, dense transforms on the minimal grid
    U x V = ceil((nu lmax + lmax_out + 1)/2) x (nu lmax + lmax_out + 1):
    2 nu C N L^2 (S1) + C [2 nu U L^2 + 2 nu U V M + (nu - 1) U V + 2 U V M_o + 2 U L_o^2] + 2 N C L_o^2 (S5)."""
    import torch
    res = []
    for (nu, lmax, N, C, batch) in [(2, 6, 64, 64, 4096), (3, 6, 64, 64, 4096), (4, 6, 64, 64, 4096),
                                    (3, 3, 32, 32, 16384), (4, 3, 32, 32, 16384)]:
        inp = synthetic.make_nbody(nu, lmax, lmax, N, C, batch, seed=0)
        # rotating input sets so that no step finds its inputs in L2
        nsets = max(2, int(300e6 // inp.X.nbytes) + 1)
        Xs = [torch.from_numpy(inp.X).to(dev) for _ in range(nsets)]
        W_in, W_out = torch.from_numpy(inp.W_in).to(dev), torch.from_numpy(inp.W_out).to(dev)
        out = torch.empty((batch, N, (lmax + 1) ** 2), device=dev)
        it = [0]

        def fn():
            it[0] += 1
            cg.cgtp_onsite_nbody(Xs[it[0] % nsets], W_in, W_out, nu, lmax, lmax, N, C, out=out)
        ms = time_steps(fn, 20, 3)
        cg.cgtp_profile_enable(True)
        for _ in range(10):
            fn()
        torch.cuda.synchronize()
        prof = cg.cgtp_profile_collect()
        cg.cgtp_profile_enable(False)
        L2 = (lmax + 1) ** 2
        U, V = (nu * lmax + lmax + 2) // 2, nu * lmax + lmax + 1
        M = 2 * lmax + 1
        core = C * (2 * nu * U * L2 + 2 * nu * U * V * M + (nu - 1) * U * V + 2 * U * V * M + 2 * U * L2)
        flops = 2 * nu * C * N * L2 + core + 2 * N * C * L2
        kms = {k: v[0] / 10 for k, v in prof.items() if v[1]}
        core_ms = kms.get("onsite_core_even", float("nan"))
        res.append({"workload": f"nu={nu} lmax=lmax_out={lmax} N=C={N} batch={batch}, grid {U}x{V}, {nsets} rotating input sets",
                    "ms_per_step": ms, "products_per_s": batch / (ms * 1e-3), "alg_tflops": flops * batch / (ms * 1e-3) / 1e12,
                    "frac_fp32_peak": flops * batch / (ms * 1e-3) / 1e12 / fp32_peak_tflops,
                    "core_alg_tflops": core * batch / (core_ms * 1e-3) / 1e12,
                    "core_frac_fp32_peak": core * batch / (core_ms * 1e-3) / 1e12 / fp32_peak_tflops,
                    "kernel_ms": kms})
        del Xs, out
        torch.cuda.empty_cache()
    return res


def run_edge_field(args, cg, synthetic, dev, fp32_peak_tflops):
    """Two feature fields, Eq.(28) on the graph of BASELINE.json configs[2]
    with an edge feature field [E, Ne, L^2] in place of R.Y.  Algorithmic flops: per edge the on-site S2-S4 work of all
    C channels plus the edge projection 2 C Ne L^2; per node 2 C N L^2 (node projection) + 2 N C L_o^2 (output)."""
    import torch
    res = []
    for (lmax, N, Ne, C, nodes, degree) in [(4, 128, 128, 128, 2048, 16), (4, 128, 8, 128, 2048, 16),
                                            (8, 128, 8, 128, 16384, 32)]:   # last: the graph of configs[4], 16 edge chunks
        m = synthetic.make_message(lmax, lmax, N, C, nodes, degree, r_max=5.0 if nodes == 2048 else 6.0, seed=0)
        XE, W_edge = synthetic.make_edge_field(m, Ne, seed=0)
        nsets = max(2, int(300e6 // XE.nbytes) + 1)   # rotating edge fields so that no step finds them in L2
        XEs = [torch.from_numpy(XE).to(dev) for _ in range(nsets)]
        t = {k: torch.from_numpy(getattr(m, k)).to(dev) for k in ("node_feats", "edge_index", "W_node", "W_out")}
        W_e = torch.from_numpy(W_edge).to(dev)
        out = torch.empty((nodes, 2, N, (lmax + 1) ** 2), device=dev)
        it = [0]

        def fn():
            it[0] += 1
            cg.cgtp_message_field(t["node_feats"], t["edge_index"], XEs[it[0] % nsets], W_e, t["W_node"], t["W_out"],
                                  lmax, lmax, N, Ne, C, m.parity_mask, out=out)
        ms = time_steps(fn, 20, 3)
        cg.cgtp_profile_enable(True)
        for _ in range(10):
            fn()
        torch.cuda.synchronize()
        prof = cg.cgtp_profile_collect()
        cg.cgtp_profile_enable(False)
        Ce = int((m.parity_mask == 0).sum())
        k = onsite_flops_per_atom(lmax, lmax, N, C, Ce, C - Ce)
        L2 = (lmax + 1) ** 2
        core = k["onsite_core_even"] + k["onsite_core_odd"]
        flops = m.E * (core + 2 * C * Ne * L2) + nodes * (2 * C * N * L2 + k["proj_out"])
        kms = {kk: v[0] / 10 for kk, v in prof.items() if v[1]}
        core_ms = kms.get("onsite_core_even", 0.0) + kms.get("onsite_core_odd", 0.0)
        # projections on tcgen05 tensor cores (3xTF32), reported beside the FP32 path, never instead of it (the rotating
        # edge-field sets hold the same values, so any two calls are comparable)
        tc = None
        try:
            cg.cgtp_set_math_mode(cg.MATH_3XTF32)
            tc_ms = time_steps(fn, 10, 3)
            torch.cuda.synchronize()
            got_tc = out.clone()
            cg.cgtp_set_math_mode(cg.MATH_FP32)
            fn()
            torch.cuda.synchronize()
            tc = {"ms_per_step": tc_ms, "edges_per_s": m.E / (tc_ms * 1e-3),
                  "max_rel_diff_vs_fp32_path": [float((got_tc[:, s_] - out[:, s_]).abs().max() / out[:, s_].abs().max())
                                                for s_ in (0, 1)]}
            del got_tc
        finally:
            cg.cgtp_set_math_mode(cg.MATH_FP32)
        res.append({"workload": f"configs[{2 if nodes == 2048 else 4}] graph ({nodes} nodes, {m.E} edges), lmax=lmax_out={lmax}, N=C={N}, edge field "
                                f"[E, {Ne}, {L2}] ({XE.nbytes / 1e6:.0f} MB, {nsets} rotating sets), half odd channels",
                    "ms_per_step": ms, "edges_per_s": m.E / (ms * 1e-3),
                    "alg_tflops": flops / (ms * 1e-3) / 1e12, "frac_fp32_peak": flops / (ms * 1e-3) / 1e12 / fp32_peak_tflops,
                    "core_alg_tflops": m.E * core / (core_ms * 1e-3) / 1e12 if core_ms else None,
                    "core_frac_fp32_peak": m.E * core / (core_ms * 1e-3) / 1e12 / fp32_peak_tflops if core_ms else None,
                    "kernel_ms": kms, "launches_per_step": int(sum(v[1] for v in prof.values()) // 10),
                    "projections_3xtf32": tc})
        del XEs, out
        torch.cuda.empty_cache()
    return res


if __name__ == "__main__":
    main()
