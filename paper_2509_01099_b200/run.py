"""Command-line driver of the ISLBM library: run a cavity, print Nu / Re, stop at the paper's steady-state criterion.

    python -m paper_2509_01099_b200.run --workload c3_1024sq --steps 20000 --every 2000
    python -m paper_2509_01099_b200.run --paper --dim 2 --points 257 --Ra 1e6 --until-steady      # Table 2
    python -m paper_2509_01099_b200.run --dim 3 --points 128 --mesh tanh --stretch 1.5 --Ra 1e6 --precision f32

Marshalling only: every step runs in the CUDA kernels behind include/islbm.h.
"""
from __future__ import annotations

import argparse
import json
import math
import time


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--workload", help="a BASELINE.json config: c1_64sq, c2_512sq, c3_1024sq, c4_128cu, c5_256cu[_uniform]")
    ap.add_argument("--paper", action="store_true", help="the paper's own mode: erf mesh Eq. 26 (a = 1.5), Ma = 0.1, T0 = T_cold")
    ap.add_argument("--dim", type=int, default=2)
    ap.add_argument("--points", type=int, default=257, help="mesh points per axis (Eq. 26 counts the two in-wall points)")
    ap.add_argument("--mesh", default="tanh", choices=["tanh", "uniform", "erf"])
    ap.add_argument("--stretch", type=float, default=1.5)
    ap.add_argument("--Ra", type=float, default=1e6)
    ap.add_argument("--Pr", type=float, default=0.71)
    ap.add_argument("--Ma", type=float, default=None, help="U / c_s (default: 0.1*sqrt(3) = BASELINE.json's U = 0.1; --paper: 0.1)")
    ap.add_argument("--T0", type=float, default=None, help="reference temperature of the buoyancy force (default 0; --paper: -0.5)")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--steps", type=int, default=10000)
    ap.add_argument("--every", type=int, default=2000, help="report (and test Eq. 30) every this many steps")
    ap.add_argument("--until-steady", action="store_true", help="stop when both residuals of Eq. 30 fall below --tol")
    ap.add_argument("--tol", type=float, default=1e-9)
    ap.add_argument("--stencil", type=int, default=0, choices=[0, 1],
                    help="0: destination-centred {j-1,j,j+1} (default); 1: upwind {j-2,j-1,j} / {j,j+1,j+2} (DESIGN.md A2)")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="islbm_set_tuning knob (repeatable), e.g. --tune shape3d=3 --tune chunk=8; results do not depend on them")
    ap.add_argument("--kernel", type=int, default=0, help="islbm_set_kernel: 0 auto, 1 generic, 2 TMA-staged, 3 uniform pure shift")
    ap.add_argument("--time", type=int, default=0, metavar="STEPS",
                    help="time islbm_step(STEPS) with CUDA events (after a warm-up of STEPS, best of 3) and print one JSON line "
                         "with us_per_step, MLUPS and the fraction of the HBM roofline; nothing else is run")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--noise", type=float, default=None, help="amplitude of the initial temperature noise (default 1e-3; --paper: 0)")
    args = ap.parse_args(argv)

    import torch
    from . import inputs, islbm

    if args.workload:
        w = inputs.workload(args.workload)
    else:
        mesh, stretch = ("erf", 1.5) if args.paper else (args.mesh, args.stretch)
        Ma = args.Ma if args.Ma is not None else (0.1 if args.paper else 0.1 * math.sqrt(3.0))
        w = inputs.custom_workload("cli", args.dim, args.points, mesh=mesh, stretch=stretch, Ra=args.Ra, Pr=args.Pr, Ma=Ma)
    T0 = args.T0 if args.T0 is not None else (-0.5 if args.paper else 0.0)
    noise = args.noise if args.noise is not None else (0.0 if args.paper else w.noise_amp)
    sim = islbm.Islbm(w.coords, w.delta, w.Ra, w.Pr, w.Ma, precision=0 if args.precision == "f64" else 1)
    sim.set_reference_temperature(T0)
    sim.set_stencil(args.stencil)
    if args.tune:
        sim.set_tuning(**{kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.tune})
    if args.kernel:
        sim.set_kernel(args.kernel)
    sim.init(args.seed, noise)
    if args.time:
        import os
        sim.step(args.time)
        torch.cuda.synchronize()
        best = float("inf")
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sim.step(args.time)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) * 1e3 / args.time)
        peak = 6650.0
        pk = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
        if os.path.exists(pk):
            with open(pk) as fh:
                peak = float(json.load(fh)["hbm_gbs"])
        bpu = (14 if sim.dim == 2 else 26) * 2 * (8 if args.precision == "f64" else 4)
        print(json.dumps({"kernel": sim.kernel_name, "tune": args.tune, "us_per_step": best, "MLUPS": sim.nodes / best,
                          "roofline_frac": sim.nodes * bpu / (best * 1e-6) / 1e9 / peak, "peak_gbs": peak}), flush=True)
        sim.close()
        return
    p = sim.params()
    print(json.dumps({"nodes": sim.nodes, "shape": sim.shape, "kernel": sim.kernel_name, "T0": T0,
                      **{k: p[k] for k in ("U", "H_lu", "nu", "alpha", "tau_f", "a_T", "dt_star")}}), flush=True)
    sim.steady_residual()
    done, t0 = 0, time.time()
    limit = args.steps if not args.until_steady else max(args.steps, 10 ** 9)
    while done < limit:
        n = min(args.every, limit - done)
        sim.step(n)
        done += n
        ru, rT = sim.steady_residual()
        d = sim.nusselt()
        d["Nu_middle"] = sim.nusselt_middle()
        d["Re_rms"] = math.sqrt(w.Ra / w.Pr * d["u2"])          # the form Tables 2 and 4 print (A22)
        torch.cuda.synchronize()
        el = time.time() - t0
        print(json.dumps({"step": done, "t_ff": done * p["dt_star"], "res_u": ru, "res_T": rT, **d,
                          "MLUPS": sim.nodes * done / el / 1e6}), flush=True)
        if args.until_steady and ru < args.tol and rT < args.tol:
            break
    sim.close()


if __name__ == "__main__":
    main()
