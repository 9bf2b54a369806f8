"""Kernel sweep of BASELINE.json configs[4]: gridder and degridder throughput at a fixed 2^26
visibilities (first 1024 baselines of the 48-station layout, 1024 timesteps, 64 channels) over
subgrid size, channels per subgrid, timesteps per subgrid and A-term interval, with forced
blocks (IDG_PLAN_FORCE_BLOCKS).  Prints a markdown table; every number is a CUDA-event time of the
stage entry point (median of `--reps`), the fraction is against the FP32 op-count roofline of
DESIGN.md section 7 and, for small blocks, the HBM byte bound is printed beside it.

    python -m paper_1909_07226_b200.sweep [--reps 3] [--quick] > profiles/<name>.md
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys

import numpy as np
import torch

from . import binding as idg
from . import synth

N_SM, LANES, HZ = 148, 128, 1.965e9


def _time(fn, reps):
    fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return float(np.median(ts))


def points(quick: bool):
    sizes = (16, 24, 32, 48)
    pts = []
    for N in sizes:
        for c in (1, 4, 16, 64):
            pts.append((N, c, 128, 256))
        for t in (32, 64, 256, 512):
            pts.append((N, 16, t, 512))
        for a in (8, 16):                      # A-term interval below the timestep limit: it caps the block
            pts.append((N, 16, 512, a))
    if quick:
        pts = [p for p in pts if p[0] in (16, 32)][::3]
    return pts


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--scalar", action="store_true", help="time the scalar (one polarisation) variant instead")
    args = ap.parse_args()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    if args.scalar:
        return scalar_report(dev, args.reps)
    hbm = 6451.2
    try:
        root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
        hbm = float(json.load(open(os.path.join(root, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        pass
    base = synth.make_workload("sweep", device=dev, identity_a=True, aterm_interval=1024)
    nvis = base.B * base.T * base.C
    print("# Kernel sweep, BASELINE.json configs[4]: %d visibilities (%d baselines x %d timesteps x %d channels), "
          "grid %d, forced blocks" % (nvis, base.B, base.T, base.C, base.params.grid_size))
    print()
    print("Command: `python -m paper_1909_07226_b200.sweep --reps %d%s`.  Times are CUDA-event medians of the stage "
          "entry points (`idg_gridder`, `idg_degridder`); roofline = 148 SMs x 128 FP32 lanes x 1.965 GHz / (18 N^2) "
          "visibilities/s; bytes bound = (32 K + 12 n_time + 96 N^2) bytes per subgrid at %.0f GB/s." %
          (args.reps, " --quick" if args.quick else "", hbm))
    print()
    print("| N | chan/subgrid | time/subgrid | K_p | subgrids | gridder ms | gridder MVis/s | frac of FP32 roofline | "
          "degridder ms | degridder MVis/s | frac | bytes-bound MVis/s |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    gen = torch.Generator(device=dev).manual_seed(1004)
    for N, c, t, a in points(args.quick):
        eff_t = min(t, a)
        n_slots = (base.T + a - 1) // a
        prm = dataclasses.replace(base.params, subgrid_size=N, kernel_size=N // 4, max_channels=c, max_timesteps=t,
                                  aterm_interval=a)
        at = 0.1 * torch.randn((n_slots, base.n_stations, N, N, 4, 2), device=dev, generator=gen)
        at[..., 0, 0] += 1.0
        at[..., 3, 0] += 1.0
        aterms = torch.view_as_complex(at)
        taper = torch.from_numpy(synth.prolate_taper(N)).to(dev)
        plan = idg.idg_plan_create(prm, base.uvw, base.freqs, base.baselines, base.n_stations)
        P, planned, skipped = plan.size()
        sub = plan.subgrids()
        out = torch.empty_like(base.vis)
        tg = _time(lambda: idg.idg_gridder(plan, base.uvw, base.vis, aterms, taper, sub), args.reps)
        td = _time(lambda: idg.idg_degridder(plan, base.uvw, sub, aterms, taper, out), args.reps)
        roof = N_SM * LANES * HZ / (18.0 * N * N)
        K = eff_t * c
        bytes_sub = 32.0 * K + 12.0 * eff_t + 96.0 * N * N
        bb = hbm * 1e9 / bytes_sub * K / 1e6
        print("| %d | %d | %d | %d | %d | %.2f | %.0f | %.3f | %.2f | %.0f | %.3f | %.0f |" %
              (N, c, eff_t, K, P, tg, planned / tg / 1e3, planned / (tg * 1e-3) / roof, td, planned / td / 1e3,
               planned / (td * 1e-3) / roof, bb))
        sys.stdout.flush()
        plan.destroy()
        del sub, out, aterms


def scalar_report(dev, reps):
    """NEXT-3: the scalar variant on the LOFAR-like and a 2000-baseline SKA-like slice, against the XU (MUFU)
    roofline 148 SMs x 16 lanes x 1.965 GHz / (2 N^2) visibilities/s and against the 4-polarisation kernels."""
    print("# Scalar (one polarisation) variant, NEXT-3")
    print()
    print("Command: `python -m paper_1909_07226_b200.sweep --scalar --reps %d`.  XU roofline = 148 x 16 x 1.965e9 / (2 N^2) vis/s." % reps)
    print()
    print("| workload | N | visibilities | scalar gridder ms | MVis/s | frac of XU roofline | scalar degridder ms | MVis/s | frac | "
          "4-pol gridder ms | 4-pol degridder ms |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for name, kw in (("lofar", {}), ("ska", dict(n_baselines=2000, baseline_offset=3000))):
        w = synth.make_workload(name, device=dev, **kw)
        N = w.params.subgrid_size
        plan = idg.idg_plan_create(w.params, w.uvw, w.freqs, w.baselines, w.n_stations)
        P, planned, _ = plan.size()
        vis_s = w.vis[..., 0].contiguous()
        gains = w.aterms[..., 0].contiguous()
        sub4 = plan.subgrids()
        sub1 = torch.view_as_complex(torch.view_as_real(sub4).reshape(-1)[: P * N * N * 2].reshape(P, N, N, 2))
        out1 = torch.empty_like(vis_s)
        out4 = torch.empty_like(w.vis)
        tg = _time(lambda: idg.idg_gridder_scalar(plan, w.uvw, vis_s, gains, w.taper, sub1), reps)
        td = _time(lambda: idg.idg_degridder_scalar(plan, w.uvw, sub1, gains, w.taper, out1), reps)
        tg4 = _time(lambda: idg.idg_gridder(plan, w.uvw, w.vis, w.aterms, w.taper, sub4), reps)
        td4 = _time(lambda: idg.idg_degridder(plan, w.uvw, sub4, w.aterms, w.taper, out4), reps)
        roof = N_SM * 16 * HZ / (2.0 * N * N)
        print("| %s | %d | %d | %.3f | %.0f | %.3f | %.3f | %.0f | %.3f | %.3f | %.3f |" %
              (name, N, planned, tg, planned / tg / 1e3, planned / (tg * 1e-3) / roof, td, planned / td / 1e3,
               planned / (td * 1e-3) / roof, tg4, td4))
        sys.stdout.flush()
        del sub1, sub4
        plan.destroy()


if __name__ == "__main__":
    main()
