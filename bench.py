#!/usr/bin/env python
"""bench.py — MLUPS / roofline fraction / WCTpDT of the ISLBM hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload NAME]
                    [--precision f64|f32] [--kernel 0..3] [--decomp replicas|slab] [--halo fused|p2p] [--no-extras]

One bench "step" is one pass of the whole hot path over one batch: LBM_PER_STEP
time steps (collide + stream/interpolate + walls)
followed by one Nusselt/Reynolds reduction (row a6).  `value` is whole-job MLUPS
(Eq. 38) with the state resident in HBM; `roofline` is the step
kernel alone (CUDA events around the islbm_step calls inside the timed region)
against the measured copy bandwidth; `e2e` is the same metric with the
pre-collision state passed in pinned HOST memory to islbm_set_populations_host
every step (the H2D copies happen inside the C-ABI call) and the diagnostics read
back to the host, serially with one handle (`e2e.serial`) and pipelined over two
handles on two streams (`e2e.pipelined`; `e2e.value` is the better of the two); `cpu_baseline` times the oracle on the host cores.  N > 1 runs
N independent cavities (one per rank, no data-path collective): weak scaling —
or, with --decomp slab, ONE cavity in slabs with the halo stored by the step
kernels into peer memory: strong scaling.  Rank 0 prints ONE JSON line.
`also` holds the other BASELINE.json configs, the uniform-mesh counterparts
(general kernel and pure-shift kernel) and the non-uniform/uniform ratios.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

LBM_PER_STEP = 20                       # LBM time steps per bench step
DEFAULT_WORKLOAD = "c5_256cu"           # 256^3 D3Q19+D3Q7 fp64, 3.5 GB per buffer >> L2: the HBM-bound config
BYTES_PER_UPDATE = {(2, 0): 224, (2, 1): 112, (3, 0): 416, (3, 1): 208}   # 2*Q*sizeof
METRIC = "MLUPS"


def dtype_name(prec, dim):
    """The arithmetic the path computes in.  fp32 storage: the stencil interpolation and the temperature collision run in
    fp32; the flow collision in fp32 in 3-D and in fp64 in 2-D."""
    if prec == 0:
        return "f64"
    if dim == 3:
        return "f32 (storage, stencil interpolation and collision)"
    return "f64 flow collision, f32 storage, stencil interpolation and temperature collision"


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def read_inst(workload, kernel, prec=0):
    """warp instructions per launch (smsp__inst_executed.sum) from the committed ncu capture, if there is one."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh).get("inst:" + f"{workload}:{kernel}" + (":f32" if prec else ""))
    return None


def read_traffic_commit():
    """commit id of the kernels the committed ncu figures were captured on (goes stale when a kernel changes)."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh).get("_commit")
    return None


def read_traffic(workload, kernel, prec=0):
    """dram bytes per launch from the committed ncu capture, if one exists for this kernel and storage precision."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh).get(f"{workload}:{kernel}" + (":f32" if prec else ""))
    return None


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_setup(n_gpus):
    """torch.distributed over NCCL when launched by torchrun; returns (rank, world, local_rank)."""
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return 0, 1, 0
    import torch.distributed as dist
    rank, local = int(os.environ["RANK"]), int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local))
    return rank, world, local


def dist_max_sum(t_local, units_local, device):
    """max over ranks of the timed duration, sum over ranks of the processed units."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return t_local, units_local
    tt = torch.tensor([t_local], dtype=torch.float64, device=device)
    uu = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    dist.all_reduce(uu, op=dist.ReduceOp.SUM)
    return tt.item(), uu.item()


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def oracle_threads():
    return max(1, len(os.sched_getaffinity(0)))


def oracle_sample(w, cores, target_seconds=2.0):
    """A bounded sample of workload w for the CPU oracle: the same mesh in x and y and the
    first nz_s z-planes (a wall-adjacent slab), sized for ~target_seconds per oracle step."""
    import numpy as np
    n = len(w.coords[0])
    per_core_mlups = 1.0 if w.dim == 3 else 1.3         # measured on this container (single thread)
    budget = int(cores * per_core_mlups * 1e6 * target_seconds)
    if w.dim == 2 or n ** 3 <= budget:
        return [np.array(c) for c in w.coords], "full mesh"
    nz_s = max(8, min(n, budget // (n * n)))
    coords = [np.array(w.coords[0]), np.array(w.coords[1]), np.array(w.coords[2][:nz_s])]
    return coords, f"x,y full ({n}x{n}), first {nz_s} z-planes of the same mesh"


def time_oracle(w, steps, warmup, cores):
    from oracle.oracle import Oracle
    coords, what = oracle_sample(w, cores)
    orc = Oracle(coords, w.delta, w.Ra, w.Pr, w.Ma, threads=cores)
    orc.init(w.seed, w.noise_amp)
    nodes = 1
    for c in coords:
        nodes *= len(c)
    for _ in range(warmup):
        orc.step(1)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.step(1)
    dt = time.perf_counter() - t0
    orc.close()
    return nodes * steps / dt / 1e6, dt / steps, what, nodes


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2509_01099_b200 import inputs
    w = inputs.workload(args.workload)
    cores = oracle_threads()
    mlups, sec_per_step, what, nodes = time_oracle(w, args.steps, args.warmup, cores)
    line = {
        "impl": "reference", "metric": METRIC, "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec_per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "nodes": w.nodes, "lattice": "D2Q9+D2Q5" if w.dim == 2 else "D3Q19+D3Q7",
                   "step": "one oracle time step on the sample"},
        "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": f"{what}; {nodes} nodes per step"},
        "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def time_device(sim, nodes, steps, warmup, lbm_per_step, flush=None):
    """K bench steps on the device; returns (seconds total, seconds inside islbm_step, launches, last Nu)."""
    import torch
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps + 2)]
    nus = []
    for _ in range(warmup):
        sim.step(lbm_per_step)
        nu = sim.nusselt()
    torch.cuda.synchronize()
    barrier()
    l0 = sim.launch_count
    ev[0].record()
    for k in range(steps):
        ev[1 + 2 * k].record()
        sim.step(lbm_per_step)
        ev[2 + 2 * k].record()
        nu = sim.nusselt()
        nus.append(nu)
    ev[-1].record()
    torch.cuda.synchronize()
    barrier()
    total = ev[0].elapsed_time(ev[-1]) * 1e-3
    in_step = sum(ev[1 + 2 * k].elapsed_time(ev[2 + 2 * k]) for k in range(steps)) * 1e-3
    # time averages over the timed window (BASELINE.json config 3; A20: plain mean of the samples)
    nu = dict(nu, Nu_hot_mean=sum(n["Nu_hot"] for n in nus) / len(nus), Re_mean=sum(n["Re"] for n in nus) / len(nus),
              u2_mean=sum(n["u2"] for n in nus) / len(nus), samples=len(nus))
    return total, in_step, sim.launch_count - l0, nu


def time_e2e(sim, state_host, steps, lbm_per_step):
    """End to end through the C-ABI with HOST buffers: every step islbm_set_populations_host copies the
    pre-collision state from pinned host memory (inside the library, on the handle's stream), then islbm_step and
    islbm_nusselt, which reads the diagnostics back to the host."""
    import torch
    f_h, g_h = state_host
    h2d = f_h.numel() * 8 + g_h.numel() * 8
    sim.set_populations_host(f_h, g_h)
    sim.step(lbm_per_step)
    sim.nusselt()
    torch.cuda.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        sim.set_populations_host(f_h, g_h)
        sim.step(lbm_per_step)
        nu = sim.nusselt()          # 7 doubles device -> host, synchronises
    e1.record()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1) * 1e-3, h2d, 56, nu


def time_e2e_pipelined(sims, state_host, steps, lbm_per_step):
    """The same end-to-end step with the copy of step k+1's inputs overlapped with the compute of step k: two handles
    (two device states) on two streams take the steps in turn.  Every step still uploads its inputs from pinned host
    memory through islbm_set_populations_host and reads its result back with islbm_nusselt, inside the timed region."""
    import torch
    f_h, g_h = state_host
    h2d = f_h.numel() * 8 + g_h.numel() * 8
    for s_ in sims:                                   # warm-up of both handles
        s_.set_populations_host(f_h, g_h)
        s_.step(lbm_per_step)
        s_.nusselt()
    torch.cuda.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sims[0].set_populations_host(f_h, g_h)
    for k in range(steps):
        cur, nxt = sims[k % 2], sims[(k + 1) % 2]
        if k + 1 < steps:
            nxt.set_populations_host(f_h, g_h)        # asynchronous on nxt's stream: overlaps cur's steps
        cur.step(lbm_per_step)
        nu = cur.nusselt()                            # device -> host, synchronises cur's stream only
    torch.cuda.synchronize()
    e1.record()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1) * 1e-3, h2d, 56, nu


def measure_workload(islbm, inputs, name, precision, steps, warmup, lbm_per_step, kernel=0):
    w = inputs.workload(name)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=precision)
    if kernel:
        sim.set_kernel(kernel)
    sim.init(w.seed, w.noise_amp)
    total, in_step, launches, nu = time_device(sim, w.nodes, steps, warmup, lbm_per_step)
    p = sim.params()
    t_lbm = in_step / (steps * lbm_per_step)
    out = {
        "mlups": w.nodes * steps * lbm_per_step / total / 1e6,
        "mlups_step_kernel_only": w.nodes / t_lbm / 1e6,
        "us_per_lbm_step": t_lbm * 1e6,
        "wctpdt_s": (total / (steps * lbm_per_step)) * p["H_lu"] / p["U"],
        "kernel": sim.kernel_name, "launches": launches, "Nu_hot": nu["Nu_hot"], "Re": nu["Re"],
        "Nu_hot_mean": nu["Nu_hot_mean"], "Re_mean": nu["Re_mean"], "nu_samples": nu["samples"],
        "Re_rms": math.sqrt(w.Ra / w.Pr * nu["u2"]), "Re_rms_mean": math.sqrt(w.Ra / w.Pr * nu["u2_mean"]),
        "total_s": total, "in_step_s": in_step, "H_lu": p["H_lu"],
    }
    return sim, w, out


def run_slab(args):
    """--decomp slab: ONE cavity decomposed into z-slabs (y-slabs in 2-D), one rank per GPU; per time step one layer
    of the planes with a velocity component along the slab axis crosses each face — stored by the step kernel itself
    into the neighbour's ghost layer over NVLink and ordered by step flags in peer memory (--halo fused, default: one
    launch per step and rank, no collective), or exchanged by torch.distributed point-to-point over NCCL after every
    step (--halo p2p) — and an all-reduce of 8 doubles per Nu/Re reduction: strong scaling.  The default
    multi-GPU mode stays `replicas` (BASELINE.json: everything runs on one GPU)."""
    import torch
    from paper_2509_01099_b200 import inputs, slab

    rank, world, local = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    prec = 0 if args.precision == "f64" else 1
    w = inputs.workload(args.workload)
    cav = slab.SlabCavity(w.coords, w.delta, w.Ra, w.Pr, w.Ma, rank, world, precision=prec, device=dev)
    cav.init(w.seed, w.noise_amp)
    if world > 1 and args.halo == "fused":
        cav.connect_ipc()      # step kernels store their boundary layers into the neighbours' ghost layers over NVLink
    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(args.warmup):
        cav.step(args.lbm_per_step)
        nu = cav.diagnostics()
    torch.cuda.synchronize()
    barrier()
    l0 = cav.sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        cav.step(args.lbm_per_step)
        nu = cav.diagnostics()
    e1.record()
    torch.cuda.synchronize()
    barrier()
    t_local = e0.elapsed_time(e1) * 1e-3
    clocks = sampler.stop() if sampler else None
    t_max, _ = dist_max_sum(t_local, 0.0, dev)
    units = float(w.nodes) * args.steps * args.lbm_per_step          # the whole cavity, processed once
    if rank == 0:
        peak, peak_src = read_peaks()
        bpu = BYTES_PER_UPDATE[(w.dim, prec)]
        p = cav.sim.params()
        line = {
            "metric": METRIC, "value": units / t_max / 1e6, "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_max / args.steps * 1e3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": dtype_name(prec, w.dim),
            "data": "synthetic",
            "config": {"workload": args.workload, "nodes_total": w.nodes, "lattice": "D2Q9+D2Q5" if w.dim == 2 else "D3Q19+D3Q7",
                       "mesh": f"{w.mesh} stretch {w.stretch}", "Ra": w.Ra, "Pr": w.Pr, "U_lu": 0.1,
                       "step": f"{args.lbm_per_step} LBM time steps (each followed by a halo exchange) + 1 Nu/Re reduction",
                       "parallelism": f"slab decomposition over {world} rank(s) along the slowest axis, 1-layer halo, "
                                      f"{'12 of 26' if w.dim == 3 else '8 of 14'} planes per face per step, halo "
                                      f"{'stored by the step kernel into peer memory (CUDA IPC), neighbours ordered by step flags in peer memory (no collective between steps)' if args.halo == 'fused' else 'by batched isend/irecv after each step'}"},
            "wctpdt_s": (t_max / (args.steps * args.lbm_per_step)) * p["H_lu"] / p["U"], "Nu_hot": nu["Nu_hot"], "Re": nu["Re"],
            "roofline": {"bound": "hbm", "achieved": bpu * w.nodes / world / (t_max / (args.steps * args.lbm_per_step)) / 1e9,
                         "peak": peak, "unit": "GB/s", "frac": bpu * w.nodes / world / (t_max / (args.steps * args.lbm_per_step)) / 1e9 / peak,
                         "traffic": None, "kernel": cav.sim.kernel_name, "peak_source": peak_src,
                         "note": "per rank, whole step including the halo exchange and the reduction"},
            "cpu_baseline": None, "e2e": None, "gpu_launches": cav.sim.launch_count - l0,
            # step kernels per LBM time step (the Nu/Re reduction adds two launches per bench step)
            "launches_per_lbm_step": (cav.sim.launch_count - l0 - 2 * args.steps) / (args.steps * args.lbm_per_step),
            "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


FULL_RUNS = (("c2_512sq", 0), ("c2_512sq_uniform", 0), ("c3_1024sq", 0), ("c3_1024sq", 1), ("c3_1024sq_uniform", 0),
             ("c4_128cu", 0), ("c5_256cu", 0), ("c5_256cu", 1), ("c5_256cu_uniform", 0))


def run_full(args):
    """--full: the step counts BASELINE.json states (configs 2-5: 20 000 / 50 000 / 5 000 / 10 000 LBM steps, the
    uniform counterparts alike), timed as ONE region per run with Nu_hot / <Re> sampled every 100 steps (DESIGN.md
    A20: plain mean of the samples over the timed window), after a 200-step warm-up.  One JSON line."""
    import torch
    from paper_2509_01099_b200 import inputs, islbm
    dev = torch.device("cuda", 0)
    peak, peak_src = read_peaks()
    out = {}
    for name, prec in FULL_RUNS:
        if args.workload not in (DEFAULT_WORKLOAD, name):       # --workload X --full: only X
            continue
        w = inputs.workload(name)
        sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=prec, device=dev)
        sim.init(w.seed, w.noise_amp)
        sim.step(200)
        sim.nusselt()
        sampler = ClockSampler(0)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nus, in_step = [], 0.0
        evs = []
        e0.record()
        for _ in range(w.steps // 100):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            sim.step(100)
            b.record()
            evs.append((a, b))
            nus.append(sim.nusselt())
        e1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        total = e0.elapsed_time(e1) * 1e-3
        in_step = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
        p = sim.params()
        bpu = BYTES_PER_UPDATE[(w.dim, prec)]
        n_lbm = (w.steps // 100) * 100
        out[name + ("_f32" if prec else "")] = {
            "lbm_steps_timed": n_lbm, "seconds": total, "mlups": w.nodes * n_lbm / total / 1e6,
            "us_per_lbm_step_kernel": in_step / n_lbm * 1e6,
            "roofline_frac": bpu * w.nodes / (in_step / n_lbm) / 1e9 / peak,
            "wctpdt_s": total / n_lbm * p["H_lu"] / p["U"], "t_ff_advanced": n_lbm * p["dt_star"], "kernel": sim.kernel_name,
            "Nu_hot_time_mean": sum(n["Nu_hot"] for n in nus) / len(nus), "Nu_hot_final": nus[-1]["Nu_hot"],
            "Re_time_mean": sum(n["Re"] for n in nus) / len(nus),
            "Re_rms_time_mean": math.sqrt(w.Ra / w.Pr * sum(n["u2"] for n in nus) / len(nus)),
            "nu_samples": len(nus), "clocks": clocks}
        sim.close()
        del sim
        torch.cuda.empty_cache()
    for nu, un in (("c2_512sq", "c2_512sq_uniform"), ("c3_1024sq", "c3_1024sq_uniform"), ("c5_256cu", "c5_256cu_uniform")):
        if nu in out and un in out:
            out[nu]["mlups_nonuniform_over_uniform"] = out[nu]["mlups"] / out[un]["mlups"]
            out[nu]["wctpdt_nonuniform_over_uniform"] = out[nu]["wctpdt_s"] / out[un]["wctpdt_s"]
    print(json.dumps({"mode": "full", "metric": METRIC, "unit": "MLUPS", "n_gpus": 1, "dtype": "f64 (keys *_f32: fp32 storage)",
                      "data": "synthetic", "peak_gbs": peak, "peak_source": peak_src,
                      "config": {"workload": "BASELINE.json configs 2-5 at their stated step counts",
                                 "sampling": "Nu_hot, <Re> every 100 steps over the timed window (DESIGN.md A20)",
                                 "uniform": "uniform counterparts through the general TMA kernel"},
                      "runs": out}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--lbm-per-step", type=int, default=LBM_PER_STEP)
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 generic, 2 TMA-staged, 3 uniform pure shift")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent cavities (weak scaling, default) or one cavity in slabs (strong scaling)")
    ap.add_argument("--halo", default="fused", choices=["fused", "p2p"],
                    help="--decomp slab: halo stored by the step kernel into peer memory (default) or exchanged with isend/irecv")
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary workloads, e2e and CPU baseline")
    ap.add_argument("--full", action="store_true",
                    help="time BASELINE.json's configs 2-5 at their stated step counts (20 000 / 50 000 / 5 000 / 10 000) "
                         "with Nu/Re sampled every 100 steps; about one minute on a B200")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.decomp == "slab":
        return run_slab(args)
    if args.full:
        return run_full(args)

    import torch
    from paper_2509_01099_b200 import inputs, islbm     # raises if libislbm.so is missing: no fallback

    rank, world, local = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    prec = 0 if args.precision == "f64" else 1
    sampler = ClockSampler(local) if rank == 0 else None
    sim, w, r = measure_workload(islbm, inputs, args.workload, prec, args.steps, args.warmup, args.lbm_per_step, args.kernel)
    clocks = sampler.stop() if sampler else None
    units = float(w.nodes) * args.steps * args.lbm_per_step
    t_max, units_sum = dist_max_sum(r["total_s"], units, dev)
    value = units_sum / t_max / 1e6

    peak, peak_src = read_peaks()
    bpu = BYTES_PER_UPDATE[(w.dim, prec)]
    t_launch = r["in_step_s"] / (args.steps * args.lbm_per_step)
    achieved = bpu * w.nodes / t_launch / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": read_traffic(args.workload, r["kernel"], prec), "traffic_commit": read_traffic_commit(),
                "kernel": r["kernel"],
                "algorithmic_bytes_per_launch": bpu * w.nodes, "bytes_per_update": bpu,
                "avg_launch_us": t_launch * 1e6, "peak_source": peak_src,
                "frac_of_nominal_8000GBs": achieved / 8000.0,      # secondary, against the nominal HBM3e figure
                "dram_bytes_per_update": (read_traffic(args.workload, r["kernel"], prec) or 0) / w.nodes or None}

    # fp32 storage is not bound by HBM (latency of the fp64 collision at 12 warps per SM, profiles/r2_c5_256cu_f32.md):
    # report the issue-slot roofline too, as the second bound it does not reach either.
    # peak = SMs x 4 warp schedulers x 1 warp instruction per clock x the maximum SM clock
    inst = read_inst(args.workload, r["kernel"], prec)
    if inst:
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        clk_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0            # the device's maximum SM clock (nvidia-smi)
        clk_hz = clk_mhz * 1e6
        roofline["alu"] = {"bound": "alu", "achieved": inst / t_launch / 1e9, "peak": sms * 4 * clk_hz / 1e9,
                           "unit": "G warp instructions/s", "frac": inst / t_launch / (sms * 4 * clk_hz),
                           "warp_instructions_per_launch": inst, "sms": sms, "sm_max_mhz": clk_mhz,
                           "frac_at_sampled_clock": (inst / t_launch / (sms * 4 * clocks["sm_mhz"] * 1e6)
                                                     if clocks and clocks.get("sm_mhz") else None),
                           "note": "issue-slot roofline; instruction count from the committed ncu capture"}

    e2e = None
    cpu = None
    extras = {}
    if not args.no_extras:
        # e2e: pre-collision state from pinned host memory, uploaded every step
        f, g = sim.get_populations()
        f_h = torch.empty(f.shape, dtype=torch.float64, pin_memory=True)
        g_h = torch.empty(g.shape, dtype=torch.float64, pin_memory=True)
        f_h.copy_(f)
        g_h.copy_(g)
        del f, g
        n_e2e = min(args.steps, 3)
        t_e2e, h2d, d2h, _ = time_e2e(sim, (f_h, g_h), n_e2e, args.lbm_per_step)
        t_e2e_max, u_e2e = dist_max_sum(t_e2e, float(w.nodes) * n_e2e * args.lbm_per_step, dev)
        e2e = {"value": u_e2e / t_e2e_max / 1e6, "unit": "MLUPS", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": n_e2e, "what": "islbm_set_populations_host (H2D of f_t,g_t from pinned host memory inside the C-ABI call) + "
                                       f"islbm_step({args.lbm_per_step}) + islbm_nusselt (D2H)"}
        # the same with a second handle on a second stream, so that the upload of step k+1 overlaps the compute of step k
        sim2 = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=prec, device=dev, stream=torch.cuda.Stream(dev))
        n_pipe = max(n_e2e, min(args.steps, 6))
        t_p, _, _, _ = time_e2e_pipelined((sim, sim2), (f_h, g_h), n_pipe, args.lbm_per_step)
        t_p_max, u_p = dist_max_sum(t_p, float(w.nodes) * n_pipe * args.lbm_per_step, dev)
        e2e["serial"] = e2e["value"]
        e2e["pipelined"] = {"value": u_p / t_p_max / 1e6, "steps": n_pipe,
                            "what": "two handles on two streams take the steps in turn: the H2D copy of step k+1 overlaps islbm_step of step k"}
        if e2e["pipelined"]["value"] > e2e["value"]:
            e2e["value"] = e2e["pipelined"]["value"]
            e2e["steps"] = n_pipe
            e2e["what"] = "pipelined over two handles on two streams (H2D of step k+1 under islbm_step of step k), each step: " + e2e["what"]
        sim2.close()
        del sim2, f_h, g_h
    sim.close()
    del sim
    torch.cuda.empty_cache()

    if not args.no_extras and rank == 0 and world == 1:
        # secondary workloads: (name, precision, kernel); kernel 0 = the library's default for that mesh,
        # 3 = the pure-shift kernel (the paper's "uniform" runs)
        for nm, pr, kn in (("c5_256cu_uniform", 0, 0), ("c5_256cu_uniform", 0, 3), ("c5_256cu", 1, 0), ("c5_256cu_uniform", 1, 3),
                           ("c3_1024sq", 0, 0), ("c3_1024sq_uniform", 0, 0), ("c3_1024sq_uniform", 0, 3), ("c3_1024sq", 1, 0),
                           ("c2_512sq", 0, 0), ("c2_512sq_uniform", 0, 0), ("c2_512sq_uniform", 0, 3), ("c4_128cu", 0, 0),
                           ("c1_64sq", 0, 0)):
            if nm == args.workload and pr == prec and kn == args.kernel:
                continue
            key = nm + ("_f32" if pr else "") + ("_shift" if kn == 3 else "")
            try:
                lps = args.lbm_per_step if "256" in nm or "128" in nm else 200
                s2, w2, r2 = measure_workload(islbm, inputs, nm, pr, max(3, args.steps // 2), 3, lps, kn)
                b2 = BYTES_PER_UPDATE[(w2.dim, pr)]
                extras[key] = {
                    "mlups": r2["mlups"], "roofline_frac": b2 * w2.nodes / (r2["us_per_lbm_step"] * 1e-6) / 1e9 / peak,
                    "us_per_lbm_step": r2["us_per_lbm_step"], "wctpdt_s": r2["wctpdt_s"], "kernel": r2["kernel"],
                    "Nu_hot_transient_mean": r2["Nu_hot_mean"], "Re_transient_mean": r2["Re_mean"],
                    "Re_rms_transient_mean": r2["Re_rms_mean"], "nu_samples": r2["nu_samples"],
                    "transient_window": f"{r2['nu_samples']} samples, one per {lps} steps from the rest + noise start",
                    "state_bytes_per_buffer": (w2.nodes * b2) // 2}
                s2.close()
                del s2
                torch.cuda.empty_cache()
            except Exception as exc:   # a secondary workload must not take the headline down
                extras[key] = {"error": str(exc)[:200]}
        # non-uniform / uniform ratios the paper reports: MLUPS ratio and WCTpDT ratio.  The
        # uniform counterpart is the FASTER of the two uniform-mesh runs (general TMA kernel on the uniform mesh, or the
        # pure-shift kernel): the ratio is not flattered by a weak denominator
        ratios = {}
        head = {"mlups": r["mlups"], "wctpdt_s": r["wctpdt_s"]}
        for nu, un in ((args.workload if prec == 0 else None, "c5_256cu_uniform"), ("c3_1024sq", "c3_1024sq_uniform"),
                       ("c2_512sq", "c2_512sq_uniform")):
            a = head if nu == args.workload else extras.get(nu)
            cands = [(k, extras[k]) for k in (un, un + "_shift") if k in extras and "mlups" in extras[k]]
            if a and cands and "mlups" in a:
                kb, b = max(cands, key=lambda kv: kv[1]["mlups"])
                ratios[nu] = {"mlups_nonuniform_over_uniform": a["mlups"] / b["mlups"],
                              "wctpdt_nonuniform_over_uniform": a["wctpdt_s"] / b["wctpdt_s"],
                              "uniform_run": kb, "uniform_kernel": b["kernel"],
                              "uniform_runs_mlups": {k: v["mlups"] for k, v in cands}}
        extras["ratios"] = ratios
        cores = oracle_threads()
        mlups_cpu, _, what, nodes_s = time_oracle(w, 3, 1, cores)
        cpu = {"value": mlups_cpu, "unit": "MLUPS", "cores": cores, "kind": "oracle",
               "sample": f"{what}; {nodes_s} nodes x 3 steps after 1 warm-up"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "MLUPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_max / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": dtype_name(prec, w.dim), "data": "synthetic",
            "config": {"workload": args.workload, "nodes_per_gpu": w.nodes, "lattice": "D2Q9+D2Q5" if w.dim == 2 else "D3Q19+D3Q7",
                       "mesh": f"{w.mesh} stretch {w.stretch}", "Ra": w.Ra, "Pr": w.Pr, "U_lu": 0.1,
                       "step": f"{args.lbm_per_step} LBM time steps + 1 Nu/Re reduction",
                       "l2": f"state {w.nodes * bpu // 2} B per buffer, two buffers, vs 126 MB L2: inputs larger than L2"
                             if w.nodes * bpu > 3e8 else "state fits in L2: fraction is not an HBM fraction",
                       "parallelism": f"{world} independent cavities (replicas, no data-path collective)"},
            "wctpdt_s": r["wctpdt_s"], "Nu_hot": r["Nu_hot"], "Re": r["Re"],
            # start-up transient out of the rest + noise state, NOT the statistic of BASELINE.json config 3 (that is
            # `bench.py --full`): mean of one sample per bench step; Re = Eq. 34 as printed (mean speed), Re_rms =
            # sqrt(Ra/Pr <u*^2>), the form the paper's tables print (A22)
            "Nu_hot_transient_mean": r["Nu_hot_mean"], "Re_transient_mean": r["Re_mean"], "Re_rms": r["Re_rms"],
            "Re_rms_transient_mean": r["Re_rms_mean"], "nu_samples": r["nu_samples"],
            "transient_window": f"{r['nu_samples']} samples, one per {args.lbm_per_step} steps, steps "
                                f"{args.warmup * args.lbm_per_step}..{(args.warmup + args.steps) * args.lbm_per_step} after the rest + noise start",
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": r["launches"], "clocks": clocks,
            "also": extras,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
