#!/usr/bin/env python
"""bench.py -- throughput of the IDG hot path on B200 (driver contract, tier-specific reading).

One "step" = one pass of the whole hot path over one synthetic workload that is resident in HBM:
Alg. 1 (V <- 0, gridder -> subgrid FFT -> adder) followed by Alg. 2 (splitter + subgrid IFFT, one fused
kernel -> degridder) with a plan made beforehand (the partition is an INPUT of both algorithms,
PAPER.md:276 / PAPER.md:315; the planner is timed separately and reported as plan_ms).
value = (visibilities gridded + visibilities degridded) / time, in MVis/s, over all ranks.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload ska|lofar|tiny|paper|sweep] [--impl reference]

Default workload: BASELINE.json configs[2] + configs[3] (SKA-low-like, 133 M visibilities), the largest
single-GPU configuration; configs[1] (LOFAR-like) is measured as a second block under "detail".
N > 1: ONE workload is sharded by baseline over the ranks (strong scaling); the timed step is Alg. 1 on the
rank's baselines -> all-reduce(SUM) of the [4][L][L] grid over NCCL -> Alg. 2 on the reduced grid.  Launched by
torch.distributed.run (one rank per GPU); a plain `python bench.py --gpus N` re-executes itself under it.
`--workload sweep` runs BASELINE.json configs[4] (gridder / degridder over subgrid size, channels, timesteps and
A-term interval) and writes a markdown table to --sweep-out.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import socket
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
# FP32 op-count roofline: 18 FP32 lane-ops (17 FMA + 1 FMUL) per (visibility, pixel);
# expressed in FLOP-equivalents at 2 per lane-op against 2 * lanes * clock.
LANE_OPS_PER_VIS_PIXEL = 18
ALU_PEAK_TFLOPS = N_SM * FP32_LANES * 2 * SM_MAX_HZ / 1e12
ALU_PEAK_SOURCE = "derived: 148 SMs x 128 FP32 lanes x 2 x 1965 MHz (DESIGN.md section 7), not in MEASURED_PEAKS.json"
HBM_FALLBACK_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures of the
# same workload (profiles/r02_ncu_summary.md); None where no capture of that workload exists.
NCU_TRAFFIC_BYTES = {
    "ska": {"gridder": int((16.009295 + 8.690905) * 1e9), "degridder": int((16.891421 + 4.243539) * 1e9),
            "subgrid_fft": None,      # ncu returned no DRAM counters for this launch (two captures); time and bytes only
            "adder": int((8.861878 + 0.119561) * 1e9), "splitter_ifft": int((0.336635 + 8.652087) * 1e9)},
}

WORKLOAD_NAMES = {
    "tiny": "configs[0] tiny: 8 stations, 32 x 10 s, 4 ch, N=24, L=256",
    "lofar": "configs[1] LOFAR-HBA-like: 48 stations (1128 baselines), 256 x 2 s, 16 ch, N=32, L=2048",
    "ska": "configs[2]+[3] SKA-low-like: 128 stations (8128 baselines), 1024 x 1 s, 16 ch, N=32, L=8192",
    "paper": "context: the paper's simulation shape (55 stations, 3122 x 10 s, 20 ch, N=48, L=2048; PAPER.md:445,471-473)",
    "sweep": "configs[4] kernel sweep: 1024 baselines x 1024 x 2 s x 64 ch = 2^26 visibilities, forced blocks",
}
SHAPES = {"tiny": (24, 256), "lofar": (32, 2048), "ska": (32, 8192), "paper": (48, 2048), "sweep": (32, 2048)}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="ska", choices=list(WORKLOAD_NAMES))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-second-block", action="store_true", help="skip the configs[1] block under detail")
    ap.add_argument("--sweep-out", default=os.path.join("gpurun_out", "sweep.md"))
    ap.add_argument("--sweep-quick", action="store_true")
    ap.add_argument("--sweep-scalar", action="store_true", help="sweep mode: time the scalar (one polarisation) variant")
    ap.add_argument("--reps", type=int, default=3, help="sweep mode: repetitions per point (median)")
    return ap.parse_args()


def config_dict(workload: str, world: int):
    """The `config` object; identical for the B200 arm and the reference arm of one (workload, N)."""
    N, L = SHAPES[workload]
    par = ("1 GPU, whole workload" if world == 1 else
           "baselines sharded over %d ranks (contiguous ranges), one NCCL all-reduce of the grid per step" % world)
    return {"workload": WORKLOAD_NAMES[workload], "subgrid_size": N, "grid_size": L, "parallelism": par,
            "l2": "fits L2" if workload == "tiny" else "inputs larger than L2 (vis + subgrids + grid > 126 MB)"}


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


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

def _oracle_pass(orc, prm, meta, d, n_baselines, model):
    """One pass of Alg. 1 + Alg. 2 over the subgrids in `meta`; returns seconds."""
    t0 = time.perf_counter()
    orc.grid(prm, meta, d["uvw"], d["freqs"], d["vis"], d["aterms"], d["taper"], grid_out=model["acc"])
    orc.degrid(prm, meta, d["uvw"], d["freqs"], model["grid"], d["aterms"], d["taper"], n_baselines)
    return time.perf_counter() - t0


def _sample_workload(workload: str):
    """A bounded, seeded SAMPLE of the workload for the oracle: the same recipe (stations, sources, A-terms, plan
    parameters) with every k-th baseline only, so that short and long baselines are both in it and nothing of the
    size of the full visibility set is ever built on the host."""
    from paper_1909_07226_b200 import synth
    stride = {"ska": 32, "paper": 16, "lofar": 4, "sweep": 16}.get(workload, 1)
    return synth.make_workload(workload, device="cpu", baseline_stride=stride), stride


def oracle_sample(workload: str, target_seconds: float):
    """Subgrids of the sampled baselines that cost about `target_seconds` of oracle time on this host."""
    from oracle import idg_oracle as orc
    w, stride = _sample_workload(workload)
    d = dict(uvw=w.uvw.numpy(), freqs=w.freqs, vis=w.vis.numpy(), aterms=w.aterms.numpy(), taper=w.taper.numpy())
    meta, planned, _ = orc.plan(w.params, d["uvw"], d["freqs"], w.baselines)
    L = w.params.grid_size
    # the model grid only has to be there: a band around the centre is filled, the rest stays zero (cheap to make)
    model = {"acc": np.zeros((4, L, L), dtype=np.complex128), "grid": np.zeros((4, L, L), dtype=np.complex128)}
    rng = np.random.default_rng(0)
    lo, hi = max(0, L // 2 - 1024), min(L, L // 2 + 1024)
    model["grid"][:, lo:hi, lo:hi] = rng.standard_normal((4, hi - lo, hi - lo)) + 1j * rng.standard_normal((4, hi - lo, hi - lo))
    probe = np.ascontiguousarray(meta[:: max(1, len(meta) // 16)][:16])
    t_probe = _oracle_pass(orc, w.params, probe, d, w.B, model)
    vis_probe = int((probe["n_time"].astype(np.int64) * probe["n_chan"]).sum())
    rate = vis_probe / max(t_probe, 1e-9)
    want = int(min(len(meta), max(16, target_seconds * rate / max(1.0, planned / len(meta)))))
    step = max(1, len(meta) // want)
    sample = np.ascontiguousarray(meta[::step][:want])
    nvis = int((sample["n_time"].astype(np.int64) * sample["n_chan"]).sum())
    what = ("%d subgrids (%d visibilities) = every %d-th subgrid of every %d-th baseline of the workload, Alg.1+Alg.2"
            % (len(sample), nvis, step, stride))
    return orc, w, d, sample, model, nvis, what


def cpu_baseline(workload: str, target_seconds=15.0):
    orc, w, d, sample, model, nvis, what = oracle_sample(workload, target_seconds)
    secs = _oracle_pass(orc, w.params, sample, d, w.B, model)
    return {"value": 2.0 * nvis / secs / 1e6, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
            "sample": "%s, %.1f s" % (what, secs)}


def run_reference(args):
    """--impl reference: the float64 oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    per_step = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    orc, w, d, sample, model, nvis, what = oracle_sample(args.workload, per_step)
    for _ in range(args.warmup):
        _oracle_pass(orc, w.params, sample, d, w.B, model)
    t = 0.0
    for _ in range(args.steps):
        t += _oracle_pass(orc, w.params, sample, d, w.B, model)
    value = 2.0 * nvis * args.steps / t / 1e6
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak" if args.gpus == 1 else "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_dict(args.workload, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                         "sample": "each step = " + what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------------------------

# one step = five kernels of this library: rows a4 + a5 run fused (idg_splitter_ifft), as inside idg_degrid
STAGES = ("zero_grid", "gridder", "subgrid_fft", "adder", "allreduce_grid", "splitter_ifft", "degridder")
KERNEL_STAGES = ("gridder", "subgrid_fft", "adder", "splitter_ifft", "degridder")


def touched_grid_pixels(meta, N, L) -> int:
    """Grid pixels covered by at least one subgrid (exact, from the plan metadata): a 2-D difference array of the
    subgrid rectangles, summed twice.  Host-side bookkeeping for the byte counts only."""
    diff = np.zeros((L + 1, L + 1), dtype=np.int32)
    np.add.at(diff, (meta["y0"], meta["x0"]), 1)
    np.add.at(diff, (meta["y0"] + N, meta["x0"]), -1)
    np.add.at(diff, (meta["y0"], meta["x0"] + N), -1)
    np.add.at(diff, (meta["y0"] + N, meta["x0"] + N), 1)
    return int(np.count_nonzero(np.cumsum(np.cumsum(diff, axis=0), axis=1)[:L, :L]))


def measure_device_steps(idg, sharding, w, plan, steps, warmup, world, dev, sampler_index=None):
    """W warm-up steps, then K timed steps (CUDA events on the launching stream).  Returns a dict of timings."""
    import torch
    import torch.distributed as dist
    L = w.params.grid_size
    sub = plan.subgrids()
    grid = torch.zeros((4, L, L), dtype=torch.complex64, device=dev)
    vis_out = torch.empty_like(w.vis)
    stream = torch.cuda.current_stream()

    def step(events=None):
        def mark(i):
            if events is not None:
                events[i].record(stream)
        mark(0)
        grid.zero_(); mark(1)                                   # Alg. 1 "V <- 0"
        idg.idg_gridder(plan, w.uvw, w.vis, w.aterms, w.taper, sub); mark(2)
        idg.idg_subgrid_fft(plan, sub, -1); mark(3)
        idg.idg_adder(plan, sub, grid); mark(4)
        if world > 1:
            sharding.allreduce_grid(grid)                       # the one exchange of the path
        mark(5)
        idg.idg_splitter_ifft(plan, grid, sub); mark(6)
        idg.idg_degridder(plan, w.uvw, sub, w.aterms, w.taper, vis_out); mark(7)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    if sampler:
        sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(STAGES) + 1)] for _ in range(steps)]
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    launches0 = idg.idg_kernel_launches()
    start.record(stream)
    for k in range(steps):
        step(evs[k])
    stop.record(stream)
    gpu_launches = idg.idg_kernel_launches() - launches0       # counted by the library at its launch sites
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    if world > 1:
        dist.barrier()
    elapsed_ms = start.elapsed_time(stop)
    stage_ms = {s: float(np.mean([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(steps)]))
                for i, s in enumerate(STAGES)}

    def _alone(fn, reps=3):    # rows a4 and a5 as separate launches (outside the timed region), for reference
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts))
    alone_ms = {"splitter": _alone(lambda: idg.idg_splitter(plan, grid, sub)),
                "subgrid_ifft": _alone(lambda: idg.idg_subgrid_fft(plan, sub, +1))}
    del grid, vis_out, sub
    return {"elapsed_ms": elapsed_ms, "stage_ms": stage_ms, "alone_ms": alone_ms, "gpu_launches": gpu_launches,
            "clocks": clocks}


def kernel_rooflines(workload, stage_ms, alone_ms, planned, P, N, touched_px, hbm, hbm_source, tensor=False,
                     tensor_dg=False):
    """Per-kernel roofline objects: achieved = ALGORITHMIC work per launch / mean launch time inside the timed
    region (36 N^2 flop-equivalents per visibility for gridder / degridder; 64 N^2 bytes per
    subgrid for the FFT; 32 N^2 bytes per subgrid + 64 (32) bytes per touched grid pixel for adder (splitter))."""
    flop_equiv = 2.0 * LANE_OPS_PER_VIS_PIXEL * float(planned) * N * N
    sub_bytes = 32.0 * N * N * P
    px = 32.0 * touched_px
    traffic = NCU_TRAFFIC_BYTES.get(workload, {})
    out = []

    def alu(name, stage):
        ach = flop_equiv / (stage_ms[stage] * 1e-3) / 1e12
        out.append({"kernel": name, "stage": stage, "bound": "alu", "achieved": ach, "peak": ALU_PEAK_TFLOPS,
                    "unit": "TFLOP/s", "frac": ach / ALU_PEAK_TFLOPS, "ms": stage_ms[stage],
                    "traffic": traffic.get(stage)})

    def mem(name, stage, nbytes, ms):
        ach = nbytes / (ms * 1e-3) / 1e9
        out.append({"kernel": name, "stage": stage, "bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s",
                    "frac": ach / hbm, "ms": ms, "algorithmic_bytes": nbytes, "traffic": traffic.get(stage),
                    "peak_source": hbm_source})

    alu("gridder_tc_kernel (tcgen05 contraction; fraction of the FP32 lane-op roofline of the direct evaluation)" if tensor
        else "gridder_kernel", "gridder")
    alu("degridder_tc_kernel (tcgen05 contraction; fraction of the FP32 lane-op roofline of the direct evaluation)"
        if tensor_dg else "degridder_kernel", "degridder")
    mem("subgrid_fft_kernel<N,fwd>", "subgrid_fft", 2 * sub_bytes, stage_ms["subgrid_fft"])
    mem("adder_kernel", "adder", sub_bytes + 2 * px, stage_ms["adder"])
    mem("subgrid_fft_kernel<N,inv,gather> (splitter + IFFT fused)", "splitter_ifft", sub_bytes + px,
        stage_ms["splitter_ifft"])
    alone = {"splitter_gbs": (sub_bytes + px) / (alone_ms["splitter"] * 1e-3) / 1e9,
             "subgrid_ifft_gbs": 2 * sub_bytes / (alone_ms["subgrid_ifft"] * 1e-3) / 1e9}
    alone["splitter_frac_of_hbm"] = alone["splitter_gbs"] / hbm
    alone["subgrid_ifft_frac_of_hbm"] = alone["subgrid_ifft_gbs"] / hbm
    return out, alone


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_1909_07226_b200 import binding as idg
    from paper_1909_07226_b200 import sharding
    from paper_1909_07226_b200 import synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    # test hooks (tests/test_gpu_bench.py): two ranks on ONE device over gloo exercise the N > 1 code path on a
    # single-GPU box; a real run uses one device per rank and NCCL
    backend = os.environ.get("IDG_BENCH_DIST_BACKEND", "nccl")
    dev_index = 0 if os.environ.get("IDG_BENCH_SINGLE_DEVICE") else local_rank
    torch.cuda.set_device(dev_index)
    dev = torch.device("cuda", dev_index)
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(backend)

    # ONE workload; rank r owns the contiguous baseline range sharding.baseline_range gives it (strong scaling).
    # The stations, sources and A-terms are drawn before the baselines are selected, so every rank sees the same
    # array, sky and Jones matrices.
    n_bl_total = len(synth.all_baselines(synth.n_stations_of(args.workload)))
    if args.workload == "sweep":
        n_bl_total = min(n_bl_total, 1024)
    b0, b1 = sharding.baseline_range(n_bl_total, world, rank)
    kw = {} if world == 1 else dict(baseline_offset=b0, n_baselines=b1 - b0)
    w = synth.make_workload(args.workload, device=dev, **kw)
    L, N = w.params.grid_size, w.params.subgrid_size
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    plan = idg.idg_plan_create(w.params, w.uvw, w.freqs, w.baselines, w.n_stations)
    plan_ms = 1e3 * (time.perf_counter() - t0)
    P, planned, skipped = plan.size()

    m = measure_device_steps(idg, sharding, w, plan, args.steps, args.warmup, world, dev, sampler_index=dev_index)
    elapsed_ms, stage_ms, clocks = m["elapsed_ms"], m["stage_ms"], m["clocks"]
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
        d_grid = torch.empty((4, L, L), dtype=torch.complex64, device=dev) if world > 1 else None
        n_e2e = max(2, min(args.steps, 5))

        def e2e_step():      # idg_grid_host ADDS into the caller's grid (Alg. 1 zeroes V once): no host memset per step
            idg.idg_grid_host(plan, h["uvw"], h["vis"], h["aterms"], h["taper"], h_grid)
            if world > 1:      # the ranks' host grids are summed through the device (NCCL has no host buffers)
                d_grid.copy_(h_grid, non_blocking=True)
                sharding.allreduce_grid(d_grid)
                h_grid.copy_(d_grid, non_blocking=True)
                torch.cuda.synchronize()
            idg.idg_degrid_host(plan, h["uvw"], h_grid, h["aterms"], h["taper"], h_out)

        def fused_step():    # one imaging cycle with the grid resident on the device; grid and visibilities come back
            idg.idg_grid_degrid_host(plan, h["uvw"], h["vis"], h["aterms"], h["taper"], h_grid, h_out)

        def time_steps(fn):
            fn()                                                # warm-up (allocates the plan's staging buffers)
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                fn()
            torch.cuda.synchronize()
            sec = (time.perf_counter() - t0) / n_e2e
            if world > 1:
                t = torch.tensor([sec], dtype=torch.float64, device=dev)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                sec = float(t.item())
            return sec

        nb = lambda x: x.numel() * x.element_size()
        two_s = time_steps(e2e_step)
        h2d = 2 * (nb(h["uvw"]) + nb(h["aterms"]) + nb(h["taper"]) + nb(h_grid)) + nb(h["vis"])
        d2h = nb(h_grid) + nb(h_out)
        if world > 1:
            h2d += nb(h_grid); d2h += nb(h_grid)
        two = {"value": 2.0 * total_vis / two_s / 1e6, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * two_s, "steps": n_e2e,
               "what": "idg_grid_host + idg_degrid_host on pinned host buffers (per rank), copies inside the timed region"}
        if world == 1:
            # the grid of one rank is the whole grid: the cycle runs as ONE call that keeps it on the device
            one_s = time_steps(fused_step)
            e2e = {"value": 2.0 * total_vis / one_s / 1e6, "unit": UNIT,
                   "h2d_bytes_per_step": int(nb(h["uvw"]) + nb(h["aterms"]) + nb(h["taper"]) + nb(h["vis"])),
                   "d2h_bytes_per_step": int(nb(h_grid) + nb(h_out)), "ms_per_step": 1e3 * one_s, "steps": n_e2e,
                   "what": "idg_grid_degrid_host on pinned host buffers: inputs up once, grid resident on the device, "
                           "grid and predicted visibilities copied back, copies inside the timed region",
                   "two_calls": two}
        else:
            e2e = two
        del h, h_grid, h_out, d_grid

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- rooflines: the dominant kernel (gridder, FP32 op-count bound) and the list of all five ----
    peaks = measured_peaks()
    hbm = float(peaks.get("hbm_gbs", HBM_FALLBACK_GBS))
    hbm_source = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback of B200_PROFILING.md"
    meta = plan.metadata()
    touched_px = touched_grid_pixels(meta, N, L)
    tensor = plan.uses_tensor_cores()
    kernels, alone = kernel_rooflines(args.workload, stage_ms, m["alone_ms"], planned, P, N, touched_px, hbm, hbm_source, tensor,
                                     plan.degridder_uses_tensor_cores())
    g = kernels[0]
    roofline = {"bound": "alu", "kernel": "gridder_tc_kernel" if tensor else "gridder_kernel", "achieved": g["achieved"], "peak": ALU_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": g["frac"], "traffic": g["traffic"], "peak_source": ALU_PEAK_SOURCE,
                "work": "18 FP32 lane-ops (17 FMA + 1 FMUL) per (visibility, pixel), 2 FLOP-equivalents each",
                "kernels": kernels}
    if clocks and clocks.get("sm_mhz"):
        roofline["frac_at_measured_clock"] = roofline["frac"] * (SM_MAX_HZ / 1e6) / clocks["sm_mhz"]
    try:     # the bare instruction mix of the inner loop, measured live (csrc/mixbench.cu): the practical ceiling
        mix = [idg.idg_bench_instruction_mix(4096, v) for v in (0, 1, 2)]
        roofline["measured_mix_peak"] = {
            "tflops": mix[0], "frac_of_alu_peak": mix[0] / ALU_PEAK_TFLOPS, "gridder_frac_of_mix_peak": g["achieved"] / mix[0],
            "what": "1 FFMA + sin/cos.approx + 8 FFMA2 per (visibility, pixel), operands as in the FP32 gridder / degridder, no global memory",
            "uniform_register_operands_tflops": mix[1], "scalar_ffma_tflops": mix[2]}
    except Exception as exc:      # reporting only
        roofline["measured_mix_peak"] = {"error": str(exc)}
    try:     # issue rate of the tensor-core kernels' MMA, measured live (csrc/mmabench.cu)
        roofline["measured_mma_cycles"] = {
            "n16_1cta": idg.idg_bench_mma_rate(16, 1), "n16_4cta": idg.idg_bench_mma_rate(16, 4),
            "n64": idg.idg_bench_mma_rate(64, 1), "n128": idg.idg_bench_mma_rate(128, 1), "n256": idg.idg_bench_mma_rate(256, 1),
            "what": "SM cycles per tcgen05.mma.cta_group::1.kind::f16 (M128 x N x K16, A in tensor memory) and SM; "
                    "the kernels use N = 16: 512 (visibility, pixel) pairs per MMA"}
    except Exception as exc:      # reporting only
        roofline["measured_mma_cycles"] = {"error": str(exc)}
    grid_bytes = 8.0 * 4 * L * L
    extra = {
        "correlations_per_s": 4.0 * value * 1e6,      # 4 polarisations per visibility (BASELINE.json's "0.5 G" reading)
        "gridder_on_tensor_cores": plan.uses_tensor_cores(),
        "degridder_on_tensor_cores": plan.degridder_uses_tensor_cores(),
        "plan_ms": plan_ms, "n_subgrids_rank0": P, "n_vis_rank0": planned, "n_vis_total": total_vis, "n_skipped_rank0": skipped,
        "stage_ms": stage_ms,
        "grid_mvis_s": planned / ((stage_ms["gridder"] + stage_ms["subgrid_fft"] + stage_ms["adder"]) * 1e-3) / 1e6,
        "degrid_mvis_s": planned / ((stage_ms["splitter_ifft"] + stage_ms["degridder"]) * 1e-3) / 1e6,
        "standalone_ms": m["alone_ms"], "standalone": alone,
        "hbm_peak_gbs": hbm, "hbm_peak_source": hbm_source, "touched_grid_pixels": touched_px,
        "collective": None if world == 1 else {
            "op": "all_reduce(SUM) of the [4][L][L] complex64 grid viewed as float32, NCCL", "bytes": grid_bytes,
            "ms": stage_ms["allreduce_grid"],
            "bus_gbs": 2.0 * (world - 1) / world * grid_bytes / (stage_ms["allreduce_grid"] * 1e-3) / 1e9},
    }
    plan.destroy()

    # ---- second block: configs[1] (LOFAR-like), same step, same kernels (detail only) ----
    if args.workload == "ska" and world == 1 and not args.no_second_block:
        del w
        torch.cuda.empty_cache()
        w2 = synth.make_workload("lofar", device=dev)
        p2 = idg.idg_plan_create(w2.params, w2.uvw, w2.freqs, w2.baselines, w2.n_stations)
        P2, planned2, _ = p2.size()
        m2 = measure_device_steps(idg, sharding, w2, p2, max(5, args.steps), args.warmup, 1, dev)
        N2, L2 = w2.params.subgrid_size, w2.params.grid_size
        k2, _ = kernel_rooflines("lofar", m2["stage_ms"], m2["alone_ms"], planned2, P2, N2,
                                 touched_grid_pixels(p2.metadata(), N2, L2), hbm, hbm_source, p2.uses_tensor_cores(),
                                 p2.degridder_uses_tensor_cores())
        ms2 = m2["elapsed_ms"] / max(5, args.steps)
        extra["configs1_lofar"] = {"workload": WORKLOAD_NAMES["lofar"], "value": 2.0 * planned2 / (ms2 * 1e-3) / 1e6,
                                   "unit": UNIT, "ms_per_step": ms2, "stage_ms": m2["stage_ms"], "kernels": k2,
                                   "note": "launch/latency-bound memory kernels at this size (35-65 us each)"}
        p2.destroy()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak" if world == 1 else "strong",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config_dict(args.workload, world),
        "clocks": clocks, "e2e": e2e, "gpu_launches": m["gpu_launches"], "roofline": roofline, "detail": extra,
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(args.workload)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs[4]: the kernel sweep (markdown table, not a bench line)
# ---------------------------------------------------------------------------------------------

def _time_call(torch, fn, reps):
    fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return float(np.median(ts))


def sweep_points(quick: bool):
    pts = []
    for N in (16, 24, 32, 48):
        for c in (1, 4, 16, 64):
            pts.append((N, c, 128, 256))
        for t in (32, 64, 256, 512):
            pts.append((N, 16, t, 512))
        for a in (8, 16):                      # A-term interval below the timestep limit: it caps the block
            pts.append((N, 16, 512, a))
    if quick:
        pts = [p for p in pts if p[0] in (16, 32)][::3]
    return pts


def run_sweep(args):
    """Gridder and degridder throughput at a fixed 2^26 visibilities over subgrid size, channels per subgrid,
    timesteps per subgrid and A-term interval, forced blocks (IDG_PLAN_FORCE_BLOCKS)."""
    import torch
    from paper_1909_07226_b200 import binding as idg
    from paper_1909_07226_b200 import synth
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    hbm = float(measured_peaks().get("hbm_gbs", HBM_FALLBACK_GBS))
    cmd = "python bench.py --workload sweep --reps %d%s%s --sweep-out <this file>" % (
        args.reps, " --sweep-quick" if args.sweep_quick else "", " --sweep-scalar" if args.sweep_scalar else "")
    os.makedirs(os.path.dirname(os.path.abspath(args.sweep_out)), exist_ok=True)
    out = open(args.sweep_out, "w")

    def emit(s=""):
        out.write(s + "\n")
        out.flush()

    fracs = []
    if args.sweep_scalar:
        emit("# Scalar (one polarisation) variant, NEXT-3")
        emit()
        emit("Command: `%s`.  XU roofline = 148 x 16 x 1.965e9 / (2 N^2) vis/s." % cmd)
        emit()
        emit("| workload | N | visibilities | scalar gridder ms | MVis/s | frac of XU roofline | scalar degridder ms | MVis/s | frac | "
             "4-pol gridder ms | 4-pol degridder ms |")
        emit("|---|---|---|---|---|---|---|---|---|---|---|")
        for name, kw in (("lofar", {}), ("ska", dict(n_baselines=2000, baseline_offset=3000))):
            w = synth.make_workload(name, device=dev, **kw)
            N = w.params.subgrid_size
            plan = idg.idg_plan_create(w.params, w.uvw, w.freqs, w.baselines, w.n_stations)
            P, planned, _ = plan.size()
            vis_s, gains = w.vis[..., 0].contiguous(), w.aterms[..., 0].contiguous()
            sub4 = plan.subgrids()
            sub1 = torch.view_as_complex(torch.view_as_real(sub4).reshape(-1)[: P * N * N * 2].reshape(P, N, N, 2))
            out1, out4 = torch.empty_like(vis_s), torch.empty_like(w.vis)
            tg = _time_call(torch, lambda: idg.idg_gridder_scalar(plan, w.uvw, vis_s, gains, w.taper, sub1), args.reps)
            td = _time_call(torch, lambda: idg.idg_degridder_scalar(plan, w.uvw, sub1, gains, w.taper, out1), args.reps)
            tg4 = _time_call(torch, lambda: idg.idg_gridder(plan, w.uvw, w.vis, w.aterms, w.taper, sub4), args.reps)
            td4 = _time_call(torch, lambda: idg.idg_degridder(plan, w.uvw, sub4, w.aterms, w.taper, out4), args.reps)
            roof = N_SM * 16 * SM_MAX_HZ / (2.0 * N * N)
            fracs += [planned / (tg * 1e-3) / roof, planned / (td * 1e-3) / roof]
            emit("| %s | %d | %d | %.3f | %.0f | %.3f | %.3f | %.0f | %.3f | %.3f | %.3f |" %
                 (name, N, planned, tg, planned / tg / 1e3, fracs[-2], td, planned / td / 1e3, fracs[-1], tg4, td4))
            del sub1, sub4
            plan.destroy()
    else:
        base = synth.make_workload("sweep", device=dev, identity_a=True, aterm_interval=1024)
        nvis = base.B * base.T * base.C
        emit("# Kernel sweep, BASELINE.json configs[4]: %d visibilities (%d baselines x %d timesteps x %d channels), "
             "grid %d, forced blocks" % (nvis, base.B, base.T, base.C, base.params.grid_size))
        emit()
        emit("Command: `%s`.  Times are CUDA-event medians of the stage entry points (`idg_gridder`, `idg_degridder`); "
             "roofline = 148 SMs x 128 FP32 lanes x 1.965 GHz / (18 N^2) visibilities/s; bytes bound = "
             "(32 K + 12 n_time + 96 N^2) bytes per subgrid at %.0f GB/s." % (cmd, hbm))
        emit()
        emit("| N | chan/subgrid | time/subgrid | K_p | subgrids | gridder ms | gridder MVis/s | frac of FP32 roofline | "
             "degridder ms | degridder MVis/s | frac | bytes-bound MVis/s |")
        emit("|---|---|---|---|---|---|---|---|---|---|---|---|")
        gen = torch.Generator(device=dev).manual_seed(1004)
        for N, c, t, a in sweep_points(args.sweep_quick):
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
            P, planned, _ = plan.size()
            sub = plan.subgrids()
            vout = torch.empty_like(base.vis)
            tg = _time_call(torch, lambda: idg.idg_gridder(plan, base.uvw, base.vis, aterms, taper, sub), args.reps)
            td = _time_call(torch, lambda: idg.idg_degridder(plan, base.uvw, sub, aterms, taper, vout), args.reps)
            roof = N_SM * FP32_LANES * SM_MAX_HZ / (18.0 * N * N)
            K = eff_t * c
            bb = hbm * 1e9 / (32.0 * K + 12.0 * eff_t + 96.0 * N * N) * K / 1e6
            fracs += [planned / (tg * 1e-3) / roof, planned / (td * 1e-3) / roof]
            emit("| %d | %d | %d | %d | %d | %.2f | %.0f | %.3f | %.2f | %.0f | %.3f | %.0f |" %
                 (N, c, eff_t, K, P, tg, planned / tg / 1e3, fracs[-2], td, planned / td / 1e3, fracs[-1], bb))
            plan.destroy()
            del sub, vout, aterms
    out.close()
    print(json.dumps({"workload": WORKLOAD_NAMES["sweep"], "table": args.sweep_out, "points": len(fracs) // 2,
                      "min_gridder_frac": min(fracs[0::2]), "min_degridder_frac": min(fracs[1::2])}))
    return 0


# ---------------------------------------------------------------------------------------------

def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` invoked plainly: re-execute under torch.distributed.run, one rank per GPU."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py --gpus %d: only %d CUDA device(s) visible" % (args.gpus, have))
    os.environ.setdefault("NCCL_DEBUG", "INFO")             # the communicator log (ranks, transports) goes to stderr
    os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        sys.exit(run_reference(a))
    if a.workload == "sweep":
        sys.exit(run_sweep(a))
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(a)
    sys.exit(run_b200(a))
