#!/usr/bin/env python
"""bench.py -- one JSON line for the PRISM hot path on N B200s (contract: task prompt / DESIGN.md).

A step = one pass of the whole hot path for one frozen-phonon configuration of the workload:
prism_build_potential -> prism_compute_smatrix -> prism_compute_output -> prism_accumulate (all section
8(a) rows).  `value` = PRISM probes/s over the whole job (all ranks), device-timed with CUDA events on the
launching stream with the library's per-kernel timing OFF; `beam_slices_per_s` is reported beside it
(BASELINE.json names both).  Per-kernel times and the roofline come from a separate, instrumented pass.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload P16|P8|P4|PR1|MS2] [--impl reference]

The default workload is BASELINE.json configs[4] (P16: 2048^2, 400 slices streamed from pinned host memory,
1201 beams, 512^2 probes), the largest single-GPU configuration; at N = 1 the line also carries short runs of
the other configurations under "other_workloads" (--no-others skips them).

N > 1 (torchrun): frozen-phonon configurations are independent problems, so rank r
takes configurations r, r+N, ... with no collective on the data path ("weak" scaling); the only
exchange is one NCCL all-reduce of the [probes][rings] sums for the phonon average.
"""
from __future__ import annotations

import argparse
import glob
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "prism_probes_per_s"
UNIT = "probes/s"
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # 148 SMs x 128 FMA lanes x 2 x 1.965 GHz
WORKLOAD_NOTE = {
    "PR1": "BASELINE.json configs[0]", "MS2": "BASELINE.json configs[1]", "P4": "BASELINE.json configs[2]",
    "P8": "BASELINE.json configs[3]", "P16": "BASELINE.json configs[4]",
}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def measured_traffic(workload: str, kernel: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of one `ncu --set full` capture of this
    kernel on this workload, from the newest profiles/rNN_traffic.csv that lists it (the .md beside each names the
    commands); None if absent."""
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv")), reverse=True):
        with open(path) as fh:
            for line in fh:
                f = [x.strip() for x in line.split(",")]
                if len(f) >= 3 and f[0] == workload and f[1] == kernel:
                    return float(f[2])
    return None


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
                getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
            }
            while not self._stop_evt.is_set():
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
                time.sleep(0.1)
        except Exception as exc:  # NVML unavailable: report that rather than invent numbers
            self.reasons.add(f"nvml_unavailable:{type(exc).__name__}")

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ oracle arm
def oracle_params(O, w):
    return O.Params(w.cell[0], w.cell[1], w.cell[2], w.nx, w.ny, w.n_slices, w.dz, w.voltage, w.alpha,
                    w.defocus, w.cs, w.f, w.det_step, w.det_max)


def oracle_sample(w, budget_s: float = 25.0):
    """Time the oracle, as it stands (unoptimised fp64 C with its own radix-2 FFT), on a bounded sample of the
    workload: whole beams (one per host thread) through the first min(S, 50) slices -- fewer only when 50 slices
    would exceed the time budget -- and 2 probes per thread on a reduced beam set; anything not run in full is
    scaled linearly in beams, slices and probes (the paper's own practice) and the result is
    marked `extrapolated`.  Returns (probes/s, description, cores, detail)."""
    import oracle as O
    cores = O.num_threads()
    p = oracle_params(O, w)
    lut_z, r_cut, lut_v = w.lut()
    atoms = w.atoms_for_phonon(0)
    beams = O.beams(p)
    n_beams, n_probes = len(beams), w.n_probes
    nb = min(n_beams, cores)
    # calibrate on one slice, then take as many slices as the budget allows, at most 50
    p1 = oracle_params(O, w.with_(n_slices=1))
    sel1 = atoms[:, 2] < w.dz
    v1 = O.potential(p1, atoms[sel1], w.z[sel1], lut_z, r_cut, lut_v)
    t0 = time.perf_counter()
    O.smatrix(p1, v1, beams[:nb])
    t_one = time.perf_counter() - t0
    s_slab = int(max(1, min(w.n_slices, 50, budget_s // max(t_one, 1e-3))))
    p_slab = oracle_params(O, w.with_(n_slices=s_slab))
    sel = atoms[:, 2] < s_slab * w.dz
    t0 = time.perf_counter()
    v = O.potential(p_slab, atoms[sel], w.z[sel], lut_z, r_cut, lut_v)
    t_pot = (time.perf_counter() - t0) * (w.n_slices / s_slab)
    # stage 1: nb whole beams through the slab, one per thread
    t0 = time.perf_counter()
    O.smatrix(p_slab, v, beams[:nb])
    t_bs = (time.perf_counter() - t0) * min(nb, cores) / (nb * s_slab)      # core-seconds per beam-slice
    t_s1 = t_bs * n_beams * w.n_slices / cores
    # stage 2: 2 probes per thread on a reduced beam set (cost is linear in beams), seeded random S-matrix
    nb2 = min(n_beams, max(4, int(2.0e9 // (w.nx * w.ny * 16))))
    rng = np.random.default_rng(1)
    s = (rng.standard_normal((nb2, w.ny, w.nx)) + 1j * rng.standard_normal((nb2, w.ny, w.nx)))
    npr = min(n_probes, cores * 2)
    t0 = time.perf_counter()
    O.prism_probes(p, s, beams[:nb2], w.probe_xy()[:npr])
    t_pr = (time.perf_counter() - t0) * min(npr, cores) / npr                # core-seconds per probe at nb2 beams
    t_s2 = t_pr * (n_beams / nb2) * n_probes / cores
    total = t_pot + t_s1 + t_s2
    extrapolated = s_slab < w.n_slices or nb < n_beams or nb2 < n_beams or npr < n_probes
    desc = (f"unoptimised fp64 oracle (plain C, own radix-2 FFT, gcc -O2, OpenMP x{cores}) on a sample of {w.name}: "
            f"potential {s_slab}/{w.n_slices} slices, {nb} whole beams x {s_slab} slices, {npr} probes x "
            f"{nb2}/{n_beams} beams; scaled linearly to {n_beams} beams x {w.n_slices} slices and {n_probes} probes")
    detail = {"potential_s": t_pot, "smatrix_s": t_s1, "output_s": t_s2, "extrapolated": bool(extrapolated),
              "beam_slices_per_s": n_beams * w.n_slices / t_s1}
    return n_probes / total, desc, cores, detail


def run_reference_multislice(args, w):
    """Oracle multislice on a bounded sample of MS2's probes (one per host thread), scaled linearly in probes."""
    import oracle as O
    cores = O.num_threads()
    p = oracle_params(O, w)
    lut_z, r_cut, lut_v = w.lut()
    t0 = time.perf_counter()
    v = O.potential(p, w.atoms_for_phonon(0), w.z, lut_z, r_cut, lut_v)
    t_pot = time.perf_counter() - t0
    xy = w.probe_xy()[:: max(1, w.n_probes // cores)][:cores]
    vals = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        O.multislice_probes(p, v, xy)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            vals.append(w.n_probes / (t_pot + dt * w.n_probes / len(xy)))
    value = float(np.mean(vals))
    desc = (f"unoptimised fp64 oracle (plain C, gcc -O2, OpenMP x{cores}): whole potential, {len(xy)} of {w.n_probes} "
            f"probes through {w.n_slices} slices, scaled linearly in probes")
    print(json.dumps({
        "impl": "reference", "metric": "multislice_probes_per_s", "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(vals), "warmup": args.warmup, "ms_per_step": 1e3 * w.n_probes / value, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{w.name} ({WORKLOAD_NOTE.get(w.name, 'test case')}): plain multislice, {w.nx}x{w.ny}, "
                               f"{w.n_slices} slices, {w.probes_x}x{w.probes_y} probes"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "extrapolated": True},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def run_reference(args):
    """--impl reference: the oracle is the reference arm for this tier (no pip-installable reference exists:
    /root/reference holds only the paper text).  Each step is one bounded sample of the workload, scaled
    linearly (`cpu_baseline.extrapolated`), so `ms_per_step` is the extrapolated time of a whole step, not the
    wall time of the sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1706_08563_b200 import workloads
    w = workloads.get(args.workload)
    if args.workload == "MS2":
        return run_reference_multislice(args, w)
    vals, last = [], None
    t_begin = time.perf_counter()
    for i in range(args.warmup + args.steps):
        # each step is one bounded sample; keep the whole run within a few minutes
        budget_left = 200.0 - (time.perf_counter() - t_begin)
        if i >= 1 and budget_left < 0 and vals:
            break
        val, desc, cores, detail = oracle_sample(w, budget_s=12.0)
        last = (desc, cores, detail)
        if i >= args.warmup or i == args.warmup + args.steps - 1 or budget_left < 60.0:
            vals.append(val)
    value = float(np.mean(vals))
    desc, cores, detail = last
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(vals), "warmup": args.warmup, "ms_per_step": 1e3 * w.n_probes / value,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "extrapolated": detail["extrapolated"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "beam_slices_per_s": detail["beam_slices_per_s"],
        "note": "ms_per_step is extrapolated from the bounded sample (steps x ms_per_step is not the wall time of this run)",
    }
    print(json.dumps(line))


def workload_config(w):
    return {"workload": f"{w.name} ({WORKLOAD_NOTE.get(w.name, 'test case')}): {w.nx}x{w.ny} grid, "
                        f"{w.n_slices} slices, f={w.f}, {w.probes_x}x{w.probes_y} probes, "
                        f"{len(w.z)} atoms, one frozen-phonon configuration per step",
            "grid": [w.nx, w.ny], "slices": w.n_slices, "f": w.f, "probes": [w.probes_x, w.probes_y],
            "atoms": int(len(w.z)), "phonons": w.n_phonons, "potential_on_host": bool(w.potential_on_host),
            "l2": "inputs larger than L2 (S-matrix and wave batch exceed 126 MB)"
                  if w.nx >= 512 else "working set fits L2; L2 flushed between steps by the workspace writes"}


# ------------------------------------------------------------------------------------------------ multislice line
def run_multislice(args, name, steps, warmup):
    """Workload MS2 (BASELINE.json configs[1], the comparison path): a step is prism_build_potential ->
    multislice_compute_output over the whole probe grid in the configuration's batches of 64 probes.  Reported as
    multislice probes/s; one GPU only."""
    import torch
    from paper_1706_08563_b200 import prism, workloads
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    w = workloads.get(name)
    p = prism.params_from_workload(w)
    lut_z, r_cut, lut_v = w.lut()
    atoms = np.ascontiguousarray(w.atoms_for_phonon(0))
    n_bins, n_probes, npix = prism.num_bins(p), w.n_probes, w.nx * w.ny
    v = torch.empty((w.n_slices, w.ny, w.nx), dtype=torch.float32, device=dev)
    out_dev = torch.empty((w.probes_y, w.probes_x, n_bins), dtype=torch.float32, device=dev)
    out_host = torch.empty((w.probes_y, w.probes_x, n_bins), dtype=torch.float32).pin_memory()
    ws = torch.empty(max(prism.workspace_bytes(p, prism.WS_POTENTIAL, len(w.z)),
                         prism.workspace_bytes(p, prism.WS_MULTISLICE)), dtype=torch.uint8, device=dev)

    def step(target):
        prism.build_potential(p, atoms, w.z, lut_z, r_cut, lut_v, v, ws)
        prism.multislice_output(p, v, target, ws)

    for _ in range(warmup):
        step(out_dev)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    prism.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step(out_dev)
    e1.record()
    torch.cuda.synchronize()
    ms_per_step = e0.elapsed_time(e1) / steps
    launches = prism.launch_count()
    clocks = sampler.stop()
    # per-kernel times come from a second, instrumented pass (a pair of events around every launch would slow
    # the timed region itself)
    prism.timing_enable(True)
    for _ in range(steps):
        step(out_dev)
    torch.cuda.synchronize()
    prism.timing_enable(False)
    kern = prism.timing_read()
    t0 = time.perf_counter()
    for _ in range(steps):
        step(out_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    hbm_peak, peak_src = measured_peaks()
    batch = w.batch if w.batch > 0 else n_probes
    band = 2.0 / 3.0 if min(w.nx, w.ny) >= 256 else 1.0                 # the in-band 2/3 of mixed space
    per_launch = 16.0 * npix * band * min(batch, n_probes)              # one pass over one batch of probes
    kernels = {}
    for kname, (ms, cnt) in kern.items():
        entry = {"ms_per_step": ms / steps, "launches_per_step": cnt / steps, "avg_ms": ms / cnt}
        if kname in ("row_step", "col_step"):
            entry["algorithmic_GBps"] = per_launch / (ms / cnt * 1e-3) / 1e9
        kernels[kname] = entry
    top = max(kernels, key=lambda n: kernels[n]["ms_per_step"])
    resident = top == "ms_resident"
    if resident:
        # one launch carries every probe through every slice with its wave in L2: bound by FP32 arithmetic
        # (N^2 (20 log2 N + 12) flop per probe-slice, nominal 5 N log2 N per line transform)
        flops = n_probes * w.n_slices * npix * (10.0 * (np.log2(w.nx) + np.log2(w.ny)) + 12.0)
        ach = flops / (kernels[top]["avg_ms"] * 1e-3) / 1e12
        roofline = {"kernel": top, "bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": ach / FP32_PEAK_TFLOPS, "traffic": measured_traffic(w.name, top),
                    "peak_source": "derived: 148 SMs x 128 lanes x 2 flop x 1.965 GHz (DESIGN.md)",
                    "note": "nominal FFT flops; an FFT is add-heavy, so one lane-operation is closer to one flop than two"}
        in_flight = f"one probe per SM in flight (resident kernel; the configuration's batch of {batch} sizes the per-pass path only)"
    else:
        ach = kernels[top].get("algorithmic_GBps", 0.0)
        roofline = {"kernel": top, "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s",
                    "frac": ach / hbm_peak, "traffic": None, "peak_source": peak_src, "bytes_per_launch": per_launch,
                    "note": "launch-sized batches: the waves of a batch stay in L2, so this is not an HBM measurement"}
        in_flight = f"in batches of {batch}"
    return {
        "metric": "multislice_probes_per_s", "value": n_probes / (ms_per_step * 1e-3), "unit": UNIT, "n_gpus": 1,
        "steps": steps, "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "complex64", "data": "synthetic",
        "config": {"workload": f"{w.name} ({WORKLOAD_NOTE.get(w.name, 'test case')}): {w.nx}x{w.ny} grid, {w.n_slices} slices, "
                               f"{w.probes_x}x{w.probes_y} probes, {in_flight}, {len(w.z)} atoms, plain multislice",
                   "l2": "the waves in flight (one 512 KB slot per SM) stay in L2; every step starts from the probe spectra"
                         if resident else
                         "a batch of 64 waves (33.5 MB) fits L2; the three-batch rotation of the timed loop does not flush it"},
        "clocks": clocks,
        "e2e": {"value": n_probes * steps / e2e_s, "unit": UNIT,
                "h2d_bytes_per_step": int(24 * len(w.z) + lut_v.size * 4 + 8 * (w.probes_x * w.nx + w.probes_y * w.ny + npix)),
                "d2h_bytes_per_step": int(out_host.numel() * 4)},
        "gpu_launches": int(launches), "launches_per_step": launches / steps,
        "roofline": roofline,
        "kernels": kernels,
    }


# ------------------------------------------------------------------------------------------------ CUDA arm
def run_prism(name, steps, warmup, world, rank, local, dist, want_cpu_baseline, slices=0):
    """The PRISM line of one workload.  Returns the JSON-able dict (on every rank; rank 0 prints it)."""
    import torch
    from paper_1706_08563_b200 import prism, sharding, workloads

    dev = torch.device("cuda", local)
    w = workloads.get(name)
    if slices > 0:                      # reduced depth, for profiler captures only (the line says so)
        w = w.with_(n_slices=slices, name=f"{w.name}-first-{slices}-slices")
    p = prism.params_from_workload(w)
    lut_z, r_cut, lut_v = w.lut()
    n_beams, n_bins, n_probes = prism.num_beams(p), prism.num_bins(p), w.n_probes
    npix = w.nx * w.ny

    # all allocations up front
    v_shape = (w.n_slices, w.ny, w.nx)
    v = (torch.empty(v_shape, dtype=torch.float32).pin_memory() if w.potential_on_host
         else torch.empty(v_shape, dtype=torch.float32, device=dev))
    s = torch.empty((n_beams, w.ny, w.nx), dtype=torch.complex64, device=dev)
    out_dev = torch.empty((w.probes_y, w.probes_x, n_bins), dtype=torch.float32, device=dev)
    out_host = torch.empty((w.probes_y, w.probes_x, n_bins), dtype=torch.float32).pin_memory()
    acc = torch.empty_like(out_dev)
    ws_bytes = max(prism.workspace_bytes(p, prism.WS_POTENTIAL, len(w.z)), prism.workspace_bytes(p, prism.WS_SMATRIX),
                   prism.workspace_bytes(p, prism.WS_OUTPUT))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
    # frozen-phonon configurations of this rank (host inputs, prepared outside the timed region)
    my_phonons = sharding.phonons_for_rank(w.n_phonons, world, rank)
    atoms = {ph: np.ascontiguousarray(w.atoms_for_phonon(ph)) for ph in my_phonons}

    def step(k, out_target):
        ph = my_phonons[k % len(my_phonons)]
        prism.build_potential(p, atoms[ph], w.z, lut_z, r_cut, lut_v, v, ws)
        beams = prism.compute_smatrix(p, v, s, ws)
        prism.compute_output(p, s, beams, out_target, ws)
        return beams

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for k in range(warmup):
        step(k, out_dev)
    barrier()

    # ---- timed region: device-resident output, CUDA events on the launching stream, library timing OFF ----
    sampler = ClockSampler(local)
    sampler.start()
    prism.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    weight = 1.0 / (steps * world)
    barrier()
    e0.record()
    for k in range(steps):
        ph = my_phonons[k % len(my_phonons)]
        stage_ev[k][0].record()
        prism.build_potential(p, atoms[ph], w.z, lut_z, r_cut, lut_v, v, ws)
        stage_ev[k][1].record()
        beams = prism.compute_smatrix(p, v, s, ws)
        stage_ev[k][2].record()
        prism.compute_output(p, s, beams, out_dev, ws)
        stage_ev[k][3].record()
        prism.accumulate(acc, out_dev, weight, first=(k == 0))          # frozen-phonon average
    sharding.all_reduce_sum(acc, dist)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = prism.launch_count()
    clocks = sampler.stop()
    stage_ms = [float(np.mean([stage_ev[k][i].elapsed_time(stage_ev[k][i + 1]) for k in range(steps)]))
                for i in range(3)]
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_per_step = ms_total / steps
    value = world * n_probes / (ms_per_step * 1e-3)

    # ---- instrumented pass: the same step with a pair of events around every launch (per-kernel table, roofline) ----
    inst_steps = max(1, min(steps, 3 if ms_per_step < 2000.0 else 1))
    prism.timing_enable(True)
    for k in range(inst_steps):
        step(k, out_dev)
    torch.cuda.synchronize()
    prism.timing_enable(False)
    kern = prism.timing_read()

    # ---- end to end: same calls, host atoms in, result delivered into pinned HOST memory inside the timed region ----
    e2e_steps = max(1, min(steps, max(3, int(90e3 / ms_per_step))))
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        step(k, out_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    # ---- comparison path: plain multislice through the same slice-step kernels ----
    # P16: BASELINE.json configs[4] names the run (64 x 64 probes on the same grid and slices); elsewhere a coarse
    # 8 x 8 sub-grid of the probe positions
    ms_n = 64 if name == "P16" else max(1, min(8, w.probes_x, w.probes_y))
    w_ms = w.with_(probes_x=ms_n, probes_y=ms_n, probe_step=(w.cell[0] / ms_n, w.cell[1] / ms_n),
                   batch=1024 if name == "P16" else w.batch)   # P16: 4 sweeps of the streamed potential
    p_ms = prism.params_from_workload(w_ms)
    del ws
    torch.cuda.empty_cache()
    out_ms = torch.empty((ms_n, ms_n, n_bins), dtype=torch.float32, device=dev)
    ws_ms = torch.empty(prism.workspace_bytes(p_ms, prism.WS_MULTISLICE), dtype=torch.uint8, device=dev)
    if name != "P16":
        prism.multislice_output(p_ms, v, out_ms, ws_ms)                  # warm-up (the P16 run is long enough without)
    barrier()
    m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m0.record()
    prism.multislice_output(p_ms, v, out_ms, ws_ms)
    m1.record()
    barrier()
    ms_probes_per_s = world * ms_n * ms_n / (m0.elapsed_time(m1) * 1e-3)
    ms_sweeps = -(-ms_n * ms_n // (w_ms.batch if w_ms.batch > 0 else ms_n * ms_n))
    del ws_ms, out_ms, s
    torch.cuda.empty_cache()
    cells = w.n_slices * (w.nx // 16) * (w.ny // 16)
    v_bytes = 4 * npix * w.n_slices if w.potential_on_host else 0
    h2d = 24 * len(w.z) + 4 * (cells + 1) + lut_v.size * 4 + v_bytes + 8 * (2 * w.nx + 2 * w.ny) \
        + 8 * n_beams * (w.probes_x + w.probes_y + 2) + 4 * (w.nx // w.f) * (w.ny // w.f)
    d2h = out_host.numel() * 4 + v_bytes
    e2e_value = world * n_probes * e2e_steps / e2e_s

    # ---- roofline of the dominant kernel (16 N^2 bytes per wave and pass; 8 N_b M^2 flop per probe) --
    hbm_peak, peak_src = measured_peaks()
    m2 = (w.nx // w.f) * (w.ny // w.f)
    # algorithmic bytes per wave and pass: mixed space is moved for the 2c in-band columns of
    # the nx only (c = prism_band_columns; whole waves below 256 points), real space in full
    # The ALGORITHMIC band is SURVEY.md 8(d)'s: the in-band 2/3 of each mixed-space row (21.3 N^2 bytes per beam-slice
    # for the two passes).  The kernels move the band rounded up to whole 32-column groups (`band_moved`, 0.6875 at
    # 2048, 0.75 at 512): those extra columns are not counted as useful bytes; fractions on the moved bytes are
    # reported beside, under "moved_band".
    banded = min(w.nx, w.ny) >= 256
    band = 2.0 / 3.0 if banded else 1.0
    band_moved = 2.0 * prism.band_columns(p) / w.nx if banded else 1.0
    mixed, real = 8 * npix * n_beams * band, 8 * npix * n_beams
    # algorithmic bytes per step and kernel class (a class may be split over several launches: the blocked layout runs
    # ROW_FINAL a few waves at a time)
    per_step_bytes = {"row_step": 2 * mixed * (w.n_slices - 1), "col_step": 2 * mixed * w.n_slices, "row_init": mixed,
                      "row_final": mixed + real}
    kernels = {}
    for kname, (ms, cnt) in kern.items():
        entry = {"ms_per_step": ms / inst_steps, "launches_per_step": cnt / inst_steps, "avg_ms": ms / cnt}
        if kname in per_step_bytes:
            entry["algorithmic_GBps"] = per_step_bytes[kname] / (ms / inst_steps * 1e-3) / 1e9
            entry["frac_of_hbm_peak"] = entry["algorithmic_GBps"] / hbm_peak
            if kname != "row_final":
                entry["frac_moved_band"] = entry["frac_of_hbm_peak"] * band_moved / band
        if kname == "beam_sum":
            # fallback for probe sets that are not a regular lattice: one CTA per probe re-reads its windows of every
            # layer (L2 / HBM): 8 N_b M^2 bytes and 8 N_b M^2 flop per probe
            entry["algorithmic_TFLOPs"] = 8.0 * n_beams * m2 * n_probes * inst_steps / (ms * 1e-3) / 1e12
            entry["window_read_GBps"] = 8.0 * n_beams * m2 * n_probes * inst_steps / (ms * 1e-3) / 1e9
            entry["frac_of_hbm_peak"] = entry["window_read_GBps"] / hbm_peak
            entry["fp32_frac"] = entry["algorithmic_TFLOPs"] / FP32_PEAK_TFLOPS
        # stage 2: the lattice kernel reads the pixel rows of a probe-row batch once and writes
        # the summed windows; window_out reads every window once
        if kname == "lattice_dft":
            sy = max(1, int(round(w.probe_step[1] / (w.cell[1] / w.ny))))
            rows_per_launch = max(1, int(round(w.probes_y * inst_steps / cnt)))
            pix_rows = min(w.ny, sy * (rows_per_launch - 1) + w.ny // w.f)
            # algorithmic: ONE read of the pixel rows the probe grid's windows cover + the summed windows written once.
            # Rows shared by consecutive probe-row batches are read again by each batch (the batch is sized by the
            # workspace): that re-read is reported as its own factor, not counted as useful bytes.
            rows_once = min(w.ny, sy * (w.probes_y - 1) + w.ny // w.f)
            rows_read = (cnt / inst_steps) * pix_rows
            lat_bytes = 8.0 * n_beams * rows_once * w.nx + 8.0 * m2 * n_probes
            entry["algorithmic_GBps"] = lat_bytes / (ms / inst_steps * 1e-3) / 1e9
            entry["frac_of_hbm_peak"] = entry["algorithmic_GBps"] / hbm_peak
            entry["batch_reread_factor"] = rows_read / rows_once
            entry["frac_incl_batch_rereads"] = ((8.0 * n_beams * rows_read * w.nx + 8.0 * m2 * n_probes)
                                                / (ms / inst_steps * 1e-3) / 1e9 / hbm_peak)
        if kname == "window_out":
            entry["algorithmic_GBps"] = 8.0 * m2 * n_probes / (ms / inst_steps * 1e-3) / 1e9
            entry["frac_of_hbm_peak"] = entry["algorithmic_GBps"] / hbm_peak
            flops2 = n_probes * m2 * 10.0 * np.log2(m2)                   # nominal 2-D FFT flops of the windows
            entry["fp32_TFLOPs_nominal"] = flops2 / (ms / inst_steps * 1e-3) / 1e12
        kernels[kname] = entry
    top = max(kernels, key=lambda n: kernels[n]["ms_per_step"])
    if top in per_step_bytes:
        ach = kernels[top]["algorithmic_GBps"]
        roofline = {"kernel": top, "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s",
                    "frac": ach / hbm_peak, "traffic": measured_traffic(w.name, top), "peak_source": peak_src,
                    "bytes_per_launch": per_step_bytes[top] / kernels[top]["launches_per_step"],
                    "bytes_assume": ("SURVEY.md 8(d): 2/3 of each mixed-space row in and out per pass "
                                     "(10.67 N^2 bytes per wave and pass)" if banded else "whole waves (grid < 256)"),
                    "moved_band": {"band_fraction": band_moved, "frac": ach / hbm_peak * band_moved / band,
                                   "bytes_per_launch": per_step_bytes[top] / kernels[top]["launches_per_step"] * band_moved / band}}
    else:
        ach = kernels[top].get("algorithmic_TFLOPs", 0.0)
        roofline = {"kernel": top, "bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": ach / FP32_PEAK_TFLOPS, "traffic": None,
                    "peak_source": "derived: 148 SMs x 128 lanes x 2 flop x 1.965 GHz (DESIGN.md)"}
    slice_ms = sum(kernels[k]["ms_per_step"] for k in ("row_init", "row_step", "col_step", "row_final") if k in kernels)
    step_bytes = 4 * mixed * w.n_slices + real                       # S row+col passes of 2 * mixed each, one real-space store
    flops = n_beams * w.n_slices * npix * (10.0 * (np.log2(w.nx) + np.log2(w.ny)) + 12.0)
    roofline["slice_step"] = {"algorithmic_GBps": step_bytes / (slice_ms * 1e-3) / 1e9,
                              "frac": step_bytes / (slice_ms * 1e-3) / 1e9 / hbm_peak,
                              "band_fraction": band, "band_fraction_moved": band_moved,
                              "unbanded_32N2_GBps": 32.0 * npix * n_beams * w.n_slices / (slice_ms * 1e-3) / 1e9,
                              "fp32_TFLOPs_nominal": flops / (slice_ms * 1e-3) / 1e12,
                              "fp32_frac": flops / (slice_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS}
    roofline["measured_in"] = (f"instrumented pass of {inst_steps} step(s) after the timed region (CUDA events around "
                               "every launch on the launching stream)")
    if w.nx == 2048 and w.ny == 2048:
        roofline["note"] = ("the two 2048-point passes take the same time; the row pass is FP32-bound (ncu: "
                            "sm__pipe_fma_cycles_active 72 %, DRAM 51 %), the column pass waits on its tile and its stores "
                            "(FMA pipe 52 %): profiles/r02_p16.md sections 3a, 3b")

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "complex64", "data": "synthetic", "config": workload_config(w), "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps},
        "gpu_launches": int(launches), "launches_per_step": launches / steps,
        "beam_slices_per_s": world * n_beams * w.n_slices / (stage_ms[1] * 1e-3),
        "stage2_probes_per_s": world * n_probes / (stage_ms[2] * 1e-3),
        "stage_ms": {"potential": stage_ms[0], "smatrix": stage_ms[1], "output": stage_ms[2]},
        "multislice": {"probes_per_s": ms_probes_per_s, "probes": ms_n * ms_n,
                       "potential_sweeps": ms_sweeps,
                       "h2d_bytes": int(ms_sweeps * v_bytes),
                       "note": "comparison path (row M1): same potential and slice-step kernels, one probe per wave; "
                               "PRISM / multislice speed-up = stage2_probes_per_s / probes_per_s once the S-matrix is built",
                       "prism_over_multislice": (world * n_probes / (ms_per_step * 1e-3)) / ms_probes_per_s},
        "roofline": roofline, "kernels": kernels,
    }
    if want_cpu_baseline and rank == 0:
        val, desc, cores, detail = oracle_sample(w, budget_s=40.0)     # whole beams through up to 50 slices
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                "extrapolated": detail["extrapolated"],
                                "beam_slices_per_s": detail["beam_slices_per_s"]}
    return line


def compact(line):
    """The keys of a full line that matter when it is reported under "other_workloads"."""
    keep = ("metric", "value", "unit", "steps", "warmup", "ms_per_step", "config", "e2e", "launches_per_step",
            "beam_slices_per_s", "stage2_probes_per_s", "stage_ms", "roofline")
    out = {k: line[k] for k in keep if k in line}
    out["config"] = {"workload": line["config"]["workload"]}
    if "kernels" in line:
        out["kernels"] = {k: {kk: vv for kk, vv in e.items() if kk in ("avg_ms", "algorithmic_GBps", "frac_of_hbm_peak")}
                          for k, e in line["kernels"].items()}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="P16", choices=["PR1", "MS2", "P4", "P8", "P16"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--slices", type=int, default=0,
                    help="run only this many slices of the workload (short runs under ncu; not a bench value)")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the short runs of the other configurations reported under other_workloads")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)

    if args.workload == "MS2":
        if rank == 0:
            print(json.dumps(run_multislice(args, "MS2", args.steps, args.warmup)))
        return

    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    line = run_prism(args.workload, args.steps, args.warmup, world, rank, local, dist,
                     want_cpu_baseline=(world == 1 and not args.no_cpu_baseline), slices=args.slices)
    if args.slices > 0:
        line["reduced"] = f"first {args.slices} slices only: a profiling run, not a measurement of the workload"
    if rank == 0 and world == 1 and args.workload == "P16" and not args.no_others and args.slices == 0:
        # the other BASELINE.json configurations, short runs on the same box (context; the line above is the headline)
        others = {}
        for other in ("P8", "P4"):
            others[other] = compact(run_prism(other, 5, 3, 1, 0, local, None, want_cpu_baseline=False))
        others["MS2"] = compact(run_multislice(args, "MS2", 5, 3))
        line["other_workloads"] = others
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
