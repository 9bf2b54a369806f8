#!/usr/bin/env python
"""bench.py -- throughput of the IDG hot path on B200 (driver contract, tier-specific reading).

One "step" = one pass of the whole hot path over one synthetic workload that is resident in HBM:
Alg. 1 (gridder -> subgrid FFT -> adder) followed by Alg. 2 (splitter + subgrid IFFT, one fused
kernel -> degridder) with a plan made beforehand (the partition is an INPUT of both algorithms,
PAPER.md:276 / PAPER.md:315; the planner is timed separately and reported as plan_ms).
value = (visibilities gridded + visibilities degridded) / time, in MVis/s, over all ranks.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload lofar|ska|tiny] [--impl reference]

N > 1 is launched by torch.distributed.run, one rank per GPU; the path shards by baseline with no
data-path collective (every rank owns a replica-sized workload: weak scaling), see DESIGN.md.
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

METRIC = "gridded+degridded MVis/s (4-pol visibilities through Alg. 1 + Alg. 2)"
UNIT = "MVis/s"
N_SM, FP32_LANES, SM_MAX_HZ = 148, 128, 1.965e9
# FP32 op-count roofline: 18 FP32 lane-ops (17 FMA + 1 FMUL) per
# (visibility, pixel); expressed in FLOP-equivalents at 2 per lane-op against 2*lanes*clock.
LANE_OPS_PER_VIS_PIXEL = 18
ALU_PEAK_TFLOPS = N_SM * FP32_LANES * 2 * SM_MAX_HZ / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum of one gridder launch from the committed ncu --set full capture
# (profiles/r01_final_ncu_summary.md); only the workload that was captured has a number
NCU_TRAFFIC_BYTES = {"lofar": 159668480 + 108218624}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="lofar", choices=["tiny", "lofar", "ska", "paper"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


WORKLOAD_NAMES = {
    "tiny": "configs[0] tiny: 8 stations, 32 x 10 s, 4 ch, N=24, L=256",
    "lofar": "configs[1] LOFAR-HBA-like: 48 stations (1128 baselines), 256 x 2 s, 16 ch, N=32, L=2048",
    "ska": "configs[2]+[3] SKA-low-like: 128 stations (8128 baselines), 1024 x 1 s, 16 ch, N=32, L=8192",
    "paper": "context: the paper's simulation shape (55 stations, 3122 x 10 s, 20 ch, N=48, L=2048; PAPER.md:445,471-473)",
}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.02)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------
# the oracle as CPU baseline (bench.py may execute oracle/ only here and in --impl reference)
# ---------------------------------------------------------------------------------------------

def _oracle_inputs(w):
    return dict(uvw=w.uvw.cpu().numpy(), freqs=w.freqs, vis=w.vis.cpu().numpy(),
                aterms=w.aterms.cpu().numpy(), taper=w.taper.cpu().numpy())


def _oracle_pass(orc, prm, meta, d, n_baselines, model):
    """One pass of Alg. 1 + Alg. 2 over the subgrids in `meta`; returns seconds."""
    t0 = time.perf_counter()
    orc.grid(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"], grid_out=model["acc"])
    orc.degrid(prm, meta, d["uvw"], d["freqs"], model["grid"], d["aterms"], d["taper"], n_baselines)
    return time.perf_counter() - t0


def oracle_sample(w, target_seconds: float):
    """Pick a bounded sample of the workload's subgrids (every k-th, so short and long baselines
    are both in it) that costs about `target_seconds` of oracle time on this host."""
    from oracle import idg_oracle as orc
    d = _oracle_inputs(w)
    meta, planned, _ = orc.plan(w.params, d["uvw"], d["freqs"], w.baselines)
    L = w.params.grid_size
    model = {"acc": np.zeros((4, L, L), dtype=np.complex128)}
    rng = np.random.default_rng(0)
    model["grid"] = (rng.standard_normal((4, L, L)) + 1j * rng.standard_normal((4, L, L)))
    probe = meta[:: max(1, len(meta) // 16)][:16]
    t_probe = _oracle_pass(orc, w.params, probe, d, w.B, model)
    vis_probe = int((probe["n_time"].astype(np.int64) * probe["n_chan"]).sum())
    rate = vis_probe / max(t_probe, 1e-9)                       # vis/s for one direction pair
    want = int(min(len(meta), max(16, target_seconds * rate / max(1.0, planned / len(meta)))))
    stride = max(1, len(meta) // want)
    sample = np.ascontiguousarray(meta[::stride][:want])
    return orc, d, sample, model, planned, len(meta)


def cpu_baseline(w, target_seconds=15.0):
    orc, d, sample, model, planned, P = oracle_sample(w, target_seconds)
    secs = _oracle_pass(orc, w.params, sample, d, w.B, model)
    nvis = int((sample["n_time"].astype(np.int64) * sample["n_chan"]).sum())
    return {"value": 2.0 * nvis / secs / 1e6, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
            "sample": "%d of %d subgrids (every %d-th), %d of %d visibilities, Alg.1+Alg.2, %.1f s"
                      % (len(sample), P, max(1, P // max(1, len(sample))), nvis, planned, secs)}


def run_reference(args):
    """--impl reference: the float64 oracle, as it stands, on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1909_07226_b200 import synth
    w = synth.make_workload(args.workload, device="cpu")
    per_step = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    orc, d, sample, model, planned, P = oracle_sample(w, per_step)
    nvis = int((sample["n_time"].astype(np.int64) * sample["n_chan"]).sum())
    for _ in range(args.warmup):
        _oracle_pass(orc, w.params, sample, d, w.B, model)
    t = 0.0
    for _ in range(args.steps):
        t += _oracle_pass(orc, w.params, sample, d, w.B, model)
    value = 2.0 * nvis * args.steps / t / 1e6
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": WORKLOAD_NAMES[args.workload]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                         "sample": "each step = %d of %d subgrids (%d of %d visibilities), Alg.1+Alg.2"
                                   % (len(sample), P, nvis, planned)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------------------------

# one step = five kernels: rows a4 + a5 run fused (idg_splitter_ifft), as inside idg_degrid
STAGES = ("gridder", "subgrid_fft", "adder", "splitter_ifft", "degridder")


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_1909_07226_b200 import binding as idg
    from paper_1909_07226_b200 import synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # every rank owns one replica-sized workload (its own realisation): weak scaling, no exchange
    w = synth.make_workload(args.workload, device=dev, seed_offset=rank)
    L, N = w.params.grid_size, w.params.subgrid_size
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    plan = idg.idg_plan_create(w.params, w.uvw, w.freqs, w.baselines, w.n_stations)
    plan_ms = 1e3 * (time.perf_counter() - t0)
    P, planned, skipped = plan.size()
    sub = plan.subgrids()
    grid = torch.zeros((4, L, L), dtype=torch.complex64, device=dev)
    vis_out = torch.empty_like(w.vis)
    stream = torch.cuda.current_stream()

    def step(events=None):
        def mark(i):
            if events is not None:
                events[i].record(stream)
        mark(0)
        idg.idg_gridder(plan, w.uvw, w.vis, w.aterms, w.taper, sub); mark(1)
        idg.idg_subgrid_fft(plan, sub, -1); mark(2)
        idg.idg_adder(plan, sub, grid); mark(3)
        idg.idg_splitter_ifft(plan, grid, sub); mark(4)
        idg.idg_degridder(plan, w.uvw, sub, w.aterms, w.taper, vis_out); mark(5)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(STAGES) + 1)] for _ in range(args.steps)]
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    launches0 = idg.idg_kernel_launches()
    start.record(stream)
    for k in range(args.steps):
        step(evs[k])
    stop.record(stream)
    gpu_launches = idg.idg_kernel_launches() - launches0      # counted by the library at its launch sites
    torch.cuda.synchronize()
    clocks = sampler.stop()
    if world > 1:
        dist.barrier()
    elapsed_ms = start.elapsed_time(stop)
    stage_ms = {s: float(np.mean([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(args.steps)]))
                for i, s in enumerate(STAGES)}
    # rows a4 and a5 on their own (outside the timed region), for their HBM fractions
    def _alone(fn, reps=3):
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))
    alone_ms = {"splitter": _alone(lambda: idg.idg_splitter(plan, grid, sub)),
                "subgrid_ifft": _alone(lambda: idg.idg_subgrid_fft(plan, sub, +1))}
    if world > 1:
        t = torch.tensor([elapsed_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        elapsed_ms = float(t.item())
        v = torch.tensor([float(planned)], dtype=torch.float64, device=dev)
        dist.all_reduce(v, op=dist.ReduceOp.SUM)
        total_vis = float(v.item())
    else:
        total_vis = float(planned)
    ms_per_step = elapsed_ms / args.steps
    value = 2.0 * total_vis / (ms_per_step * 1e-3) / 1e6

    # ---- end to end through the host-buffer C-ABI calls (pinned host memory, copies timed) ----
    e2e = None
    if not args.no_e2e:
        h = {k: getattr(w, k).cpu().pin_memory() for k in ("uvw", "vis", "aterms", "taper")}
        h_grid = torch.zeros((4, L, L), dtype=torch.complex64).pin_memory()
        h_out = torch.empty(w.vis.shape, dtype=torch.complex64).pin_memory()
        n_e2e = max(2, min(args.steps, 5))
        idg.idg_grid_host(plan, h["uvw"], h["vis"], h["aterms"], h["taper"], h_grid)      # warm-up (allocates staging)
        idg.idg_degrid_host(plan, h["uvw"], h_grid, h["aterms"], h["taper"], h_out)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            idg.idg_grid_host(plan, h["uvw"], h["vis"], h["aterms"], h["taper"], h_grid)
            idg.idg_degrid_host(plan, h["uvw"], h_grid, h["aterms"], h["taper"], h_out)
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / n_e2e
        if world > 1:
            t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_s = float(t.item())
        nb = lambda x: x.numel() * x.element_size()
        h2d = 2 * (nb(h["uvw"]) + nb(h["aterms"]) + nb(h["taper"]) + nb(h_grid)) + nb(h["vis"])
        d2h = nb(h_grid) + nb(h_out)
        e2e = {"value": 2.0 * total_vis / e2e_s / 1e6, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * e2e_s, "steps": n_e2e,
               "what": "idg_grid_host + idg_degrid_host on pinned host buffers, copies inside the timed region"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel: the gridder (FP32 op-count bound) --------------------
    vis_pixels = float(planned) * N * N
    flop_equiv = 2.0 * LANE_OPS_PER_VIS_PIXEL * vis_pixels
    ach = flop_equiv / (stage_ms["gridder"] * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "gridder_kernel", "achieved": ach, "peak": ALU_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": ach / ALU_PEAK_TFLOPS, "traffic": NCU_TRAFFIC_BYTES.get(args.workload),
                "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1965 MHz (DESIGN.md), not in MEASURED_PEAKS.json",
                "work": "18 FP32 lane-ops (17 FMA + 1 FMUL) per (visibility, pixel), 2 FLOP-equivalents each"}
    if clocks.get("sm_mhz"):
        roofline["frac_at_measured_clock"] = roofline["frac"] * (SM_MAX_HZ / 1e6) / clocks["sm_mhz"]
    ach_d = flop_equiv / (stage_ms["degridder"] * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    sub_bytes = 32.0 * N * N * P
    # grid pixels covered by at least one subgrid (exact, from the plan metadata): a 2-D difference array
    # of the subgrid rectangles, summed twice.  Host-side bookkeeping for the byte count only.
    meta = plan.metadata()
    diff = np.zeros((L + 1, L + 1), dtype=np.int32)
    np.add.at(diff, (meta["y0"], meta["x0"]), 1)
    np.add.at(diff, (meta["y0"] + N, meta["x0"]), -1)
    np.add.at(diff, (meta["y0"], meta["x0"] + N), -1)
    np.add.at(diff, (meta["y0"] + N, meta["x0"] + N), 1)
    touched_px = int(np.count_nonzero(np.cumsum(np.cumsum(diff, axis=0), axis=1)[:L, :L]))
    touched = 2 * 32.0 * touched_px                      # read + write of every touched 4-pol grid pixel
    extra = {
        "correlations_per_s": 4.0 * value * 1e6,      # 4 polarisations per visibility (BASELINE.json's "0.5 G" reading)
        "plan_ms": plan_ms, "n_subgrids": P, "n_vis_per_rank": planned, "n_skipped": skipped,
        "stage_ms": stage_ms,
        "grid_mvis_s": planned / ((stage_ms["gridder"] + stage_ms["subgrid_fft"] + stage_ms["adder"]) * 1e-3) / 1e6,
        "degrid_mvis_s": planned / ((stage_ms["splitter_ifft"] + stage_ms["degridder"]) * 1e-3) / 1e6,
        "standalone_ms": alone_ms,     # idg_splitter and idg_subgrid_fft(+1) as separate launches, untimed region
        "degridder_roofline_frac": ach_d / ALU_PEAK_TFLOPS,
        "adder_gbs": (sub_bytes + touched) / (stage_ms["adder"] * 1e-3) / 1e9,
        "splitter_gbs": (sub_bytes + touched / 2) / (alone_ms["splitter"] * 1e-3) / 1e9,
        "splitter_ifft_gbs": (sub_bytes + touched / 2) / (stage_ms["splitter_ifft"] * 1e-3) / 1e9,
        "subgrid_fft_gbs": 2 * sub_bytes / (stage_ms["subgrid_fft"] * 1e-3) / 1e9,
        "hbm_peak_gbs": hbm, "hbm_peak_source": "measured" if peaks else "fallback",
        "touched_grid_pixels": touched_px,
        "adder_frac_of_hbm": (sub_bytes + touched) / (stage_ms["adder"] * 1e-3) / 1e9 / hbm,
        "splitter_frac_of_hbm": (sub_bytes + touched / 2) / (alone_ms["splitter"] * 1e-3) / 1e9 / hbm,
        "splitter_ifft_frac_of_hbm": (sub_bytes + touched / 2) / (stage_ms["splitter_ifft"] * 1e-3) / 1e9 / hbm,
        "subgrid_fft_frac_of_hbm": 2 * sub_bytes / (stage_ms["subgrid_fft"] * 1e-3) / 1e9 / hbm,
    }
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAMES[args.workload], "subgrid_size": N, "grid_size": L,
                   "parallelism": "baselines sharded, %d replica(s), no collective" % world,
                   "l2": "inputs larger than L2 (vis + subgrids + grid > 126 MB)" if args.workload != "tiny" else "fits L2"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": gpu_launches, "roofline": roofline, "detail": extra,
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(w.to("cpu"))
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse_args()
    sys.exit(run_reference(a) if a.impl == "reference" else run_b200(a))
