#!/usr/bin/env python
"""bench.py -- throughput of the SDM coalescence hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl reference]

One "step" = one pass of the whole hot path (rows a1-a8 of DESIGN.md) over the resident state:
    sdm_remove_zero -> sdm_coalescence_step_moments (coalescence step + global moments of the new state).
Default workload: C5 of BASELINE.json (512x512 cells x 256 droplets = 2^26 super-droplets,
gravitational kernel), the configuration the >= 60 % HBM-roofline target is quoted on; it is 1.25 GiB
of state, far larger than the 126 MB L2, so no L2 flush is needed between iterations.

Prints ONE JSON line (rank 0).  N > 1 (under torchrun): every rank runs its own shard of cells on
its own GPU -- cells are independent, there is no data-path collective -- weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "super-droplet-steps/s"
UNIT = "sd-steps/s"

# algorithmic bytes per droplet-step: compulsory traffic of the method
B_ALG_FUSED_KERNEL = 24.0      # dominant kernel, cell-contiguous path: read xi 8 + v 8 + cell_id 4, write idx 4
B_ALG_STEP = 24.0              # the whole step: the same 24 B (the cell index of the next step is derived inside the
                               # dominant kernel; moments ride on the same pass; remove_zero: 0 when nothing to remove)


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


# committed ncu captures that roofline.traffic is read from, and the kernel sources each one describes (the contract test
# fails when a source file has a later commit than its capture)
TRAFFIC_SOURCES = {"C5": "r03_ncu_fused_kernel_c5.csv", "C5s": "r02_ncu_general_path_c5s.csv"}
TRAFFIC_KERNEL_SOURCES = {"C5": ("sdm_fused_count.cuh", "sdm_fused.cuh"), "C5s": ("sdm_general.cuh",)}


def ncu_dram_bytes(path):
    """dram__bytes_read.sum + dram__bytes_write.sum of the first captured launch in an ncu summary csv."""
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    total, seen = 0.0, 0
    try:
        with open(path) as f:
            for line in f:
                parts = line.strip().split(",")
                if parts[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    total += float(parts[2]) * scale[parts[1]]
                    seen += 1
    except Exception:
        return None
    return total if seen == 2 else None


def build_workload(name: str, rank: int = 0, scale_cells: int | None = None):
    import workloads
    if name == "C5":
        nx = ny = scale_cells or 512
        return workloads.grid_uniform(nx, ny, 256, seed=rank), f"C5: {nx}x{ny} cells x 256 droplets, gravitational kernel, cell-contiguous"
    if name == "C5s":
        nx = ny = scale_cells or 512
        return (workloads.grid_uniform(nx, ny, 256, seed=rank, shuffled=True),
                f"C5s: {nx}x{ny} cells x 256 droplets, gravitational kernel, SHUFFLED storage (as after displacement)")
    if name == "C5d":
        nx = ny = scale_cells or 512
        w = workloads.grid_uniform(nx, ny, 256, seed=rank)
        w.dV = 1.0                                 # collision-dense: p ~ 2.6e-2 per pair, the screening flags most cells
        return w, f"C5d: {nx}x{ny} cells x 256 droplets, gravitational kernel, dV = 1 (collision-dense), cell-contiguous"
    if name == "C4x":                              # C4 at HBM scale: 1024x1024 cells of ~64 droplets (2^26), small cells in groups
        return (workloads.grid_poisson(1024, 1024, 64.0, shuffled=False, seed=rank),
                "C4x: 1024x1024 cells, Poisson(64)/cell (6.7e7 droplets), Golovin, cell-contiguous")
    if name == "C5m":                              # C5 with 64 droplets per cell: 1024x1024 cells x 64
        return (workloads.grid_uniform(1024, 1024, 64, seed=rank),
                "C5m: 1024x1024 cells x 64 droplets, gravitational kernel, cell-contiguous")
    if name == "C4":
        return workloads.grid_poisson(shuffled=False, seed=rank), "C4: 128x128 cells, Poisson(64)/cell, Golovin, cell-contiguous"
    if name == "C4s":
        return workloads.grid_poisson(shuffled=True, seed=rank), "C4: 128x128 cells, Poisson(64)/cell, Golovin, shuffled storage"
    if name == "C1":
        return workloads.golovin_box(2 ** 13), "C1: Golovin box n=2^13"
    if name == "C2a":
        return workloads.golovin_box(2 ** 17), "C2: Golovin box n=2^17"
    if name == "C2b":
        return workloads.golovin_box(2 ** 20), "C2: Golovin box n=2^20"
    if name == "C3":
        return workloads.gravitational_box(2 ** 20), "C3: gravitational box n=2^20"
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """SM clocks and throttle reasons sampled DURING the timed region (B200_PROFILING.md): an NVML polling thread that
    reads the SM clock back to back (no sleep: a 6.5 ms region of 20 C5 steps still gets tens of samples) and the
    throttle reasons and the board power on every fourth pass."""

    REASONS = (("hw_slowdown", "nvmlClocksEventReasonHwSlowdown"),
               ("hw_thermal_slowdown", "nvmlClocksEventReasonHwThermalSlowdown"),
               ("sw_thermal_slowdown", "nvmlClocksEventReasonSwThermalSlowdown"),
               ("sw_power_cap", "nvmlClocksEventReasonSwPowerCap"))

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.sm, self.power, self.bits, self.max_mhz = [], [], 0, None
        self.stop_flag = threading.Event()
        self.thread = None
        self.error = None

    def _handle(self, nv):
        import torch
        try:                                       # CUDA_VISIBLE_DEVICES may renumber devices: go by UUID
            uuid = str(torch.cuda.get_device_properties(self.gpu).uuid)
            return nv.nvmlDeviceGetHandleByUUID(("GPU-" + uuid).encode())
        except Exception:
            return nv.nvmlDeviceGetHandleByIndex(self.gpu)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv, self.h = nv, self._handle(nv)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
            # the first call of each query can take milliseconds (lazy initialisation inside NVML): make it here, not in
            # the polling thread, or a 6.5 ms timed region is over before the first sample arrives
            nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
            nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            nv.nvmlDeviceGetPowerUsage(self.h)
        except Exception as e:                     # noqa: BLE001
            self.error = f"NVML unavailable: {e}"
            return
        self.thread = threading.Thread(target=self._poll, daemon=True)
        self.thread.start()
        t0 = time.perf_counter()                   # return once the thread is polling (bounded wait)
        while not self.sm and self.error is None and time.perf_counter() - t0 < 0.5:
            time.sleep(0.0002)

    def _poll(self):
        nv = self.nv
        k = 0
        while not self.stop_flag.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                if k % 4 == 0:
                    self.bits |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                    self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception as e:                 # noqa: BLE001
                self.error = str(e)
                return
            k += 1
            if len(self.sm) >= 200000:             # a seconds-long region: thin out instead of growing without bound
                time.sleep(0.0005)

    def stop(self):
        if self.thread is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": [self.error or "not started"]}
        self.stop_flag.set()
        self.thread.join(timeout=5)
        reasons = [name for name, attr in self.REASONS if self.bits & int(getattr(self.nv, attr, 0))]
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "sm_mhz_min": min(self.sm) if self.sm else None,
                "power_w": statistics.median(self.power) if self.power else None,
                "power_w_max": max(self.power) if self.power else None,
                "samples": len(self.sm), "reasons": reasons}


def cpu_info():
    """CPU model string and core count of the box the oracle is timed on (SURVEY.md 8(d) "Oracle timing")."""
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return model, os.cpu_count()


def oracle_sample_rate(target_s: float = 12.0, full: bool = False, full_workload=None):
    """The oracle as it stands, one thread: three steps of the full-size C5 state for the default workload (about 40 s
    of CPU work; SURVEY.md 8(d) "Oracle timing"), a bounded C5-shaped sample (64x64 cells x 256) otherwise."""
    import oracle
    import workloads
    if full:
        w = full_workload if full_workload is not None else workloads.grid_uniform(512, 512, 256, seed=0)
    else:
        w = workloads.grid_uniform(64, 64, 256, seed=0)
    if full:
        target_s = 1e9
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    steps, t0 = 0, time.perf_counter()
    while True:
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, steps, want_perm=True)
        oracle.moments(xi, v)
        steps += 1
        el = time.perf_counter() - t0
        if el >= target_s or steps >= (3 if full else 200):
            break
    return w.n_sd * steps / el, steps, w.n_sd, el


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores (bounded sample per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    import workloads
    w = workloads.grid_uniform(64, 64, 256, seed=0)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()

    def one(step):
        nonlocal xi, v, cell
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        oracle.moments(xi, v)

    for s in range(args.warmup):
        one(s)
    t0 = time.perf_counter()
    for s in range(args.steps):
        one(args.warmup + s)
    el = time.perf_counter() - t0
    value = w.n_sd * args.steps / el
    model, nproc = cpu_info()
    sample = f"C5-shaped sample: 64x64 cells x 256 droplets (2^20) per step, single thread on {model} ({nproc} cores)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "C5: 512x512 cells x 256 droplets, gravitational kernel (reference arm runs a bounded sample)",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "cpu_model": model, "nproc": nproc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="sdm", choices=["sdm", "reference"])
    ap.add_argument("--workload", default="C5")
    ap.add_argument("--cells", type=int, default=None, help="C5 only: grid edge (default 512)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-baseline-full", action="store_true",
                    help="time the oracle on 3 steps of the full-size C5 state instead of the 2^20 sample (~1 min)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sustained", action="store_true", help="skip the seconds-long steady-state region after the headline")
    ap.add_argument("--sustained-seconds", type=float, default=3.0,
                    help="full-size C5 on one GPU: length of the steady-state region timed after the headline region")
    ap.add_argument("--e2e-serial", action="store_true", help="e2e on ONE handle: H2D, step, D2H strictly one after the other")
    ap.add_argument("--e2e-shards", type=int, default=8, help="cell-range shards of the pipelined e2e measurement")
    ap.add_argument("--per-step-calls", action="store_true",
                    help="box workloads: time sdm_remove_zero + sdm_coalescence_step_moments per step instead of one sdm_run")
    ap.add_argument("--lanes", type=int, default=0, help="tuning: lanes per cell of the fused kernel (0 = auto)")
    ap.add_argument("--ctas-per-sm", type=int, default=0, help="tuning: grid of the counting-sort kernel (0 = auto)")
    ap.add_argument("--box-ctas", type=int, default=0, help="tuning: CTAs of the persistent box kernel (0 = auto)")
    ap.add_argument("--engine", type=int, default=0, help="tuning: per-cell sort engine (0 auto, 1 network, 2 bucket)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    import numpy as np
    import torch
    import paper_2101_06318_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libsdm has no CPU fallback")
    pkg.load_library()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w, wname = build_workload(args.workload, rank, args.cells)
    dev = torch.device("cuda", local)
    s = pkg.SDM(w.n_sd, w.n_cell, device=dev)
    hx = torch.from_numpy(w.xi).pin_memory()
    hv = torch.from_numpy(w.v).pin_memory()
    hc = torch.from_numpy(w.cell_id).pin_memory()
    s.set_state_host(hx, hv, hc)
    s.set_option(pkg.OPT_TIMING, 1)
    if args.lanes:
        s.set_option(pkg.OPT_LANES_PER_CELL, args.lanes)
    if args.engine:
        s.set_option(pkg.OPT_SORT_ENGINE, args.engine)
    if args.ctas_per_sm:
        s.set_option(pkg.OPT_CTAS_PER_SM, args.ctas_per_sm)
    if args.box_ctas:
        s.set_option(pkg.OPT_BOX_CTAS, args.box_ctas)
    mode = s.counters()["mode"]

    from paper_2101_06318_b200 import sharding
    # N > 1: rank r holds cells [r, r+1) / N of ONE global state (weak scaling: every rank the same number of cells):
    # same Philox seed everywhere, global storage indices through the index base (sdm_set_index_base), and the three
    # global moments all-gathered and summed on the device inside every timed step.  Boxes (one cell) do not shard:
    # replicas with their own seeds.
    seed = w.seed if mode != 2 else sharding.shard_seed(w.seed, rank)
    if mode != 2 and world > 1:
        s.set_index_base(rank * w.n_sd)          # no multiplicity can reach zero in this workload (checked after the run)
    dmom = sharding.DeviceMoments(dev, world)
    mom = dmom.out

    def one_step(step):
        s.remove_zero(sync=False)
        s.coalescence_step_moments(w.dt, w.dV, w.kernel, w.kparam, seed, step, out=mom)
        if world > 1:
            dmom.reduce()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # single-cell boxes (C1-C3): the paper's own benchmark is the 3600-step loop, which the library
    # runs as ONE sdm_run call -- [remove_zero; step] x K inside one persistent launch -- followed by the moments
    box_run = mode == 2 and not args.per_step_calls

    def timed_steps(first, count):
        if box_run:
            s.run(w.dt, w.dV, w.kernel, w.kparam, seed, first, count, True)
            s.moments(out=mom)
        else:
            for st in range(count):
                one_step(first + st)

    timed_steps(0, args.warmup)
    barrier()
    s.timing()                                   # drop warm-up kernel timings
    launches0 = s.counters()["launches"]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    timed_steps(args.warmup, args.steps)
    ev1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = ev0.elapsed_time(ev1)
    kernel_ms, kernel_n = s.timing()
    cnt = s.counters()
    if world > 1 and mode != 2 and cnt["n_sd"] != w.n_sd:
        raise SystemExit("a shard lost droplets: the index bases would have had to be re-derived (sharding.rebase)")
    launches = cnt["launches"] - launches0
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    value = world * w.n_sd * args.steps / (ms * 1e-3)

    # Steady state (MEASURED_PEAKS.json distinguishes burst from sustained): the headline region of the driver's
    # --steps 20 is a 6.5 ms burst at ~260 W; over seconds the board reaches its power cap and the SM clock drops.  So
    # the full-size C5 run goes on for >= --sustained-seconds more, timed the same way (CUDA events around the whole
    # region, the library's own events around every launch of the dominant kernel), clocks sampled throughout.
    sustained = None
    if args.workload == "C5" and args.cells is None and world == 1 and mode == 1 and not args.no_sustained:
        batch = 3000                               # sdm_get_timing keeps at most 4096 launches between two calls
        n_batches = max(1, int(round(args.sustained_seconds * 1e3 / max(ms / args.steps, 1e-3) / batch)))
        sus_sampler = ClockSampler(local)
        sus_sampler.start()
        sk_ms, sk_n, first = 0.0, 0, args.warmup + args.steps
        sv0, sv1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        sv0.record()
        for b in range(n_batches):
            timed_steps(first + b * batch, batch)
            k_ms, k_n = s.timing()                 # synchronises: one host round trip per 3000 steps (~1 s)
            sk_ms, sk_n = sk_ms + k_ms, sk_n + k_n
        sv1.record()
        torch.cuda.synchronize()
        sus_clocks = sus_sampler.stop()
        sus_ms = sv0.elapsed_time(sv1)
        sustained = {"steps": n_batches * batch, "seconds": sus_ms * 1e-3, "ms_per_step": sus_ms / (n_batches * batch),
                     "kernel_ms": sk_ms / max(sk_n, 1), "launches_timed": sk_n,
                     "sm_mhz_median": sus_clocks.get("sm_mhz"), "sm_mhz_min": sus_clocks.get("sm_mhz_min"),
                     "power_w_median": sus_clocks.get("power_w"), "power_w_max": sus_clocks.get("power_w_max"),
                     "clock_samples": sus_clocks.get("samples"), "reasons": sus_clocks.get("reasons")}
        cnt = s.counters()

    # end to end through the C ABI with HOST buffers: H2D of the state, the step, D2H of the state
    e2e = None
    if not args.no_e2e:
        ox = torch.empty(w.n_sd, dtype=torch.int64).pin_memory()
        ov = torch.empty(w.n_sd, dtype=torch.float64).pin_memory()
        oc = torch.empty(w.n_sd, dtype=torch.int32).pin_memory()

        def e2e_step(step):
            s.set_state_host(hx, hv, hc)
            one_step(step)
            return s.get_state_host(ox, ov, oc)

        what = "sdm_set_state_host + remove_zero + coalescence_step_moments + sdm_get_state_host, pinned host buffers"
        pipe = None
        if mode == 1 and w.n_cell >= 64 and not args.e2e_serial:
            # Cells are independent and the Philox counter is the global storage index (sdm_set_index_base), so the same
            # calls on K cell-range shards -- one handle, one stream and one host thread each -- give the same result
            # while H2D of shard k+1 overlaps the step and the D2H of shard k (both copy engines busy).
            import concurrent.futures
            K = args.e2e_shards
            counts = np.bincount(w.cell_id, minlength=w.n_cell)
            parts = [p for p in sharding.partition_cells(counts, K) if p.sd_hi > p.sd_lo]
            shards = []
            for p in parts:
                sl = slice(p.sd_lo, p.sd_hi)
                lc = torch.from_numpy((w.cell_id[sl] - p.cell_lo).astype(np.int32)).pin_memory()
                hs = pkg.SDM(p.sd_hi - p.sd_lo, p.cell_hi - p.cell_lo, device=dev, stream=torch.cuda.Stream(dev))
                hs.set_index_base(rank * w.n_sd + p.sd_lo if world > 1 else p.sd_lo)
                mo = (torch.empty(1, dtype=torch.int64, device=dev), torch.empty(1, dtype=torch.float64, device=dev),
                      torch.empty(1, dtype=torch.float64, device=dev))
                shards.append((hs, sl, lc, mo))
            pool = concurrent.futures.ThreadPoolExecutor(max_workers=len(shards))

            def shard_step(args_):
                (hs, sl, lc, m), step = args_
                with torch.cuda.stream(hs.stream):
                    hs.set_state_host(hx[sl], hv[sl], lc)
                    hs.remove_zero(sync=False)
                    hs.coalescence_step_moments(w.dt, w.dV, w.kernel, w.kparam, seed, step, out=m)
                    return hs.get_state_host(ox[sl], ov[sl], oc[sl])

            def e2e_step(step):                    # noqa: F811 -- the pipelined variant replaces the serial one
                return sum(pool.map(shard_step, [(sh, step) for sh in shards]))

            pipe = len(shards)
            what = (f"the same calls on {pipe} cell-range shards (own handle, stream and host thread each; global storage "
                    "indices through sdm_set_index_base): H2D, step and D2H of different shards overlap")
        n_back = e2e_step(0)
        assert n_back == w.n_sd, (n_back, w.n_sd)
        barrier()
        t0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for st in range(args.e2e_steps):
            e2e_step(1 + st)
        e1.record()
        barrier()
        wall = time.perf_counter() - t0
        ems = max(e0.elapsed_time(e1), wall * 1e3)
        if pipe is not None:
            for hs, _, _, _ in shards:
                hs.close()
            pool.shutdown()
        if dist is not None:
            t = torch.tensor([ems], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ems = float(t.item())
        e2e = {"value": world * w.n_sd * args.e2e_steps / (ems * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": 20 * w.n_sd, "d2h_bytes_per_step": 20 * w.n_sd + 8,
               "steps": args.e2e_steps, "ms_per_step": ems / args.e2e_steps,
               "what": what}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peak, peak_src = measured_peak_gbs()
    roofline = None
    if kernel_n > 0:
        per_launch_s = kernel_ms * 1e-3 / kernel_n
        b_alg = B_ALG_FUSED_KERNEL if mode == 1 else None
        if b_alg is not None:
            achieved = b_alg * w.n_sd / per_launch_s / 1e9
            roofline = {"bound": "hbm", "kernel": "k_fused_cells_count (TMA staging, Philox, per-cell counting sort, pairs, update, moments, next cell table from cell_id)",
                        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                        "traffic": None, "peak_source": peak_src, "ms_per_launch": per_launch_s * 1e3,
                        "launches_timed": kernel_n, "alg_bytes_per_droplet": b_alg,
                        "kernel_share_of_step": kernel_ms / ms if ms > 0 else None,
                        "whole_step": {"alg_bytes_per_droplet": B_ALG_STEP,
                                       "achieved": B_ALG_STEP * w.n_sd * args.steps / (ms * 1e-3) / 1e9,
                                       "frac": B_ALG_STEP * w.n_sd * args.steps / (ms * 1e-3) / 1e9 / peak}}
            if sustained is not None:
                # same algorithmic bytes, same peak: the fraction the kernel / the whole step keeps over seconds
                sustained["frac"] = b_alg * w.n_sd / (sustained["kernel_ms"] * 1e-3) / 1e9 / peak
                sustained["whole_step_frac"] = B_ALG_STEP * w.n_sd / (sustained["ms_per_step"] * 1e-3) / 1e9 / peak
                roofline["sustained"] = sustained
        else:
            # general path (any storage order) and box path: the same 24 algorithmic bytes per droplet-step; what the
            # gathers and scattered stores of shuffled storage cost on top counts against the implementation
            whole = B_ALG_STEP * w.n_sd * args.steps / (ms * 1e-3) / 1e9
            hbm_resident = 20 * w.n_sd > 2 * 126e6
            roofline = {"bound": "hbm", "kernel": ("k_box_steps (persistent box kernel; L2-resident workload)" if mode == 2
                                                   else "k_segment_sort_pairs (general path: sort + pairs of one segment per warp)"),
                        "achieved": whole if hbm_resident else None, "peak": peak, "unit": "GB/s",
                        "frac": whole / peak if hbm_resident else None, "traffic": None,
                        "what": ("whole step (all launches of the general path) at 24 algorithmic bytes per droplet"
                                 if hbm_resident else "L2-resident workload: no HBM roofline applies"),
                        "peak_source": peak_src, "alg_bytes_per_droplet": B_ALG_STEP,
                        "ms_per_launch": per_launch_s * 1e3, "launches_timed": kernel_n,
                        "kernel_share_of_step": kernel_ms / ms if ms > 0 else None}
    # traffic: DRAM bytes (read + write) per launch of the dominant kernel, from the committed ncu capture of this
    # command (not measured in this run: a profiler is never attached to a timed run)
    if roofline is not None and w.n_sd == 67108864:
        src = TRAFFIC_SOURCES.get(args.workload)
        if src is not None:
            roofline["traffic"] = ncu_dram_bytes(os.path.join(ROOT, "profiles", src))
            roofline["traffic_source"] = "profiles/" + src + " (ncu --set full capture of the same command)"

    cpu = None
    if not args.no_cpu_baseline:
        # three steps of the full-size C5 state whatever --steps is (SURVEY.md 8(d) "Oracle timing": C5, >= 3 steps;
        # ~36 s of one host core); the 2^20-droplet sample for reduced grids and the other workloads
        full = args.cpu_baseline_full or (args.workload == "C5" and args.cells is None)
        rate, osteps, on, oel = oracle_sample_rate(full=full, full_workload=w if args.workload == "C5" and args.cells is None else None)
        model, nproc = cpu_info()
        shape = "full C5 state: 512x512" if full else "C5-shaped sample: 64x64"
        cpu = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "cpu_model": model, "nproc": nproc,
               "sample": f"{shape} cells x 256 droplets (n_sd={on}), {osteps} steps in {oel:.1f} s, single thread"}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "n_sd_per_gpu": w.n_sd, "n_cell_per_gpu": w.n_cell,
                   "step": ("one sdm_run(K steps, remove_zero each step) + sdm_moments: all K steps in one persistent launch"
                            if box_run else "sdm_remove_zero + sdm_coalescence_step_moments (step + global moments)"),
                   "path": {0: "general", 1: "fused cell-contiguous", 2: "single-cell box (persistent cooperative kernel)"}[mode],
                   "l2": "inputs larger than L2 (no flush)" if 20 * w.n_sd > 2 * 126e6 else "L2-resident workload (no flush; latency/launch-bound)",
                   "parallelism": (f"cells sharded over {world} GPU(s) (one global state, same seed, index bases); no data-path "
                                   "collective; global moments all-gathered (24 B per rank) and summed on the device every step"
                                   if mode != 2 else f"{world} independent replica(s) of the box (own seeds)")},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
        "events_in_run": cnt["events"],
    }
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
