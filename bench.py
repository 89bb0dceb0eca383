"""bench.py - throughput of the graph-based SP2 density-matrix path (arXiv:1603.00937) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload water4096] [--impl ours|reference]

One STEP = one pass of the whole hot path over one synthetic system (rows 0-6):
gbe_build_graph (bounds, S_tau, halos, D pattern) + gbe_density (gather, 40 SP2 iterations with the on-device
branch choice, core-column scatter).  Metric: density-matrix orbitals/s = orbitals / step time.

* `value`   : inputs resident in HBM, step timed with CUDA events on the launching stream.
* `e2e`     : the same step through the C ABI's HOST entry points (gbe_build_graph_host + gbe_density_host):
              H comes from pinned host memory and D goes back to pinned host memory inside the timed region.
* `roofline`: the dominant kernel (k_x2, FP64 tensor pipe), per-launch time from CUDA events recorded around every
              launch by gbe_density_timed in the same process.
* `cpu_baseline` / `--impl reference`: the CPU oracle as it stands, on a bounded sample of the same workload.

N > 1 (torchrun): the path does not shard across GPUs in this build (north_star: one GPU, no collectives) - every rank
runs an independent replica on its own seeded system ("replicas only"); value = all orbitals / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "density_matrix_orbitals_per_s"
UNIT = "orbitals/s"
# FP64 tensor ceiling.  MEASURED_PEAKS.json has no FP64 entry and the profiling guide states no nominal FP64
# figure, so the ceiling is MEASURED IN THIS RUN, before the timed region, the way the driver measures bf16: cuBLAS DGEMM
# (torch.matmul, float64, 8192^3), best of 10 (burst) and back to back for 4 s (sustained) -> roofline.peak.  Beside it:
# the DMMA issue rate = 128 flop/clk/SM (one DMMA.8x8x4 = 512 flop per 16 cycles per SM sub-partition, measured in
# profiles/r01_fp64_peak_probe.md) x SM count x the SM clock sampled during the timed region.
DMMA_FLOP_PER_CLK_PER_SM = 128.0
HBM_NOMINAL_GBS = 8000.0  # north_star: "about 8 TB/s"
X2_TRAFFIC_JSON = os.path.join(ROOT, "profiles", "x2_traffic.json")
X2_SOURCE = os.path.join(ROOT, "paper_1603_00937_b200", "csrc", "gbe_x2.cu")
# one oracle pass over the 4,096-molecule box takes about 28 s on the box's 16 host cores (BENCH_r01)
ORACLE_S_PER_MOLECULE_16_CORES = 28.0 / 4096

WORKLOADS = {
    # name: (molecules, communities) - BASELINE.json configs[1], configs[2] (SURVEY numbering: config 2, config 3)
    "water1024": (1024, 128),
    "water4096": (4096, 512),
    # BASELINE.json configs[3]: 2,000-residue random coil in water, ~1.2e5 orbitals, heterogeneous core+halo sizes
    "peptide2000": (None, None),
}


def make_system(workload: str, seed: int):
    import gbe_inputs as gi
    if workload == "peptide2000":
        return gi.peptide_water(2000, seed=seed)
    n_mol, n_part = WORKLOADS[workload]
    return gi.water_box(n_mol, n_part, seed=seed)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tf=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    source="MEASURED_PEAKS.json (of measured)")
    return dict(hbm_gbs=6650.0, bf16_tf=1400.0, source="B200_PROFILING.md fallback (of fallback)")


def git_blob_sha1(path: str) -> str:
    """The git blob hash of a file's current content (what `git hash-object` prints)."""
    import hashlib
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def x2_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_x2 launch from the tracked ncu record - only if that record
    was captured on this workload AND on the gbe_x2.cu that is being run now (git blob hash); else None."""
    try:
        with open(X2_TRAFFIC_JSON) as f:
            rec = json.load(f)
    except (OSError, ValueError):
        return None, "no profiles/x2_traffic.json"
    if rec.get("workload") != workload:
        return None, "profiles/x2_traffic.json was captured on workload %r" % rec.get("workload")
    if rec.get("gbe_x2_cu_blob") != git_blob_sha1(X2_SOURCE):
        return None, "profiles/x2_traffic.json was captured on another version of gbe_x2.cu (blob %s)" % rec.get("gbe_x2_cu_blob")
    return float(rec["dram_bytes_per_launch"]), "B per launch, dram read + write, %s" % rec.get("source", "ncu --set full")


def record_traffic(args) -> None:
    """--record-traffic RAW.csv: reads an `ncu -i ... --page raw --csv` export of a `--set full` capture of k_x2 on this
    workload and writes profiles/x2_traffic.json (mean over the captured full-size launches), stamped with the git blob
    hash of the gbe_x2.cu in the tree."""
    import csv
    rows = list(csv.reader(open(args.record_traffic)))
    hdr = rows[0]
    k_name, k_rd, k_wr, k_grid = (hdr.index(c) for c in ("Kernel Name", "dram__bytes_read.sum", "dram__bytes_write.sum", "Grid Size"))
    unit_rd, unit_wr = rows[1][k_rd], rows[1][k_wr]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    per = []
    for r in rows[2:]:
        if "k_x2" in r[k_name]:
            per.append((int(r[k_grid].strip("()").split(",")[0]),
                        float(r[k_rd].replace(",", "")) * scale[unit_rd] + float(r[k_wr].replace(",", "")) * scale[unit_wr]))
    assert per, "no k_x2 launch in the capture"
    full = max(g for g, _ in per)
    vals = [b for g, b in per if g == full]
    kname = next(r[k_name] for r in rows[2:] if "k_x2" in r[k_name]).split("(")[0].replace("void ", "").replace("<unnamed>::", "")
    rec = {"workload": args.workload, "kernel": kname, "grid": full, "launches_averaged": len(vals),
           "dram_bytes_per_launch": float(np.mean(vals)), "gbe_x2_cu_blob": git_blob_sha1(X2_SOURCE),
           "source": args.traffic_source or os.path.basename(args.record_traffic)}
    with open(X2_TRAFFIC_JSON, "w") as f:
        json.dump(rec, f, indent=1)
        f.write("\n")
    print(json.dumps(rec))


def measure_fp64_peak(torch) -> dict:
    """cuBLAS DGEMM in this process, after the timed regions (a library call, used for the roofline denominator only):
    torch.matmul on float64 8192^3, best of 10 (burst) and back to back for ~4 s (sustained), CUDA events."""
    n = 8192
    a = torch.randn(n, n, dtype=torch.float64, device="cuda")
    b = torch.randn(n, n, dtype=torch.float64, device="cuda")
    c = torch.empty(n, n, dtype=torch.float64, device="cuda")
    flop = 2.0 * n ** 3
    for _ in range(2):
        torch.matmul(a, b, out=c)
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b, out=c)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    reps = max(10, int(4000.0 / best))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        torch.matmul(a, b, out=c)
    e1.record()
    torch.cuda.synchronize()
    sustained = e0.elapsed_time(e1) / reps
    del a, b, c
    torch.cuda.empty_cache()
    return {"burst_tflops": flop / (best * 1e-3) * 1e-12, "sustained_tflops": flop / (sustained * 1e-3) * 1e-12,
            "reps_sustained": reps}


CLOCK_REASONS = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]


def _clock_summary(rows, t0: float, t1: float, source: str) -> dict:
    """rows: (wall time, sm MHz, max sm MHz, power W, set of reason names); the samples inside [t0, t1] summarised."""
    sm, smax, pw, reasons = [], [], [], set()
    for ts, a, b, c, r in rows:
        if t0 <= ts <= t1 + 0.2:
            sm.append(a); smax.append(b); pw.append(c); reasons |= r
    return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
            "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons), "source": source}


class NvmlSampler:
    """SM clock, power and throttle reasons through NVML from a thread of this process, every 50 ms.  The default: a
    separate nvidia-smi process takes a driver lock when it attaches, polls and exits, and each of those showed up as a
    stall of tens of ms in a timed step; NVML queries from inside the process did not."""

    def __init__(self, gpu_index: int):
        import pynvml
        self.nv = pynvml
        pynvml.nvmlInit()
        # NVML numbers every device of the box, CUDA those of CUDA_VISIBLE_DEVICES: translate the index when it is set
        vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
        ids = [x.strip() for x in vis.split(",") if x.strip()]
        if ids and gpu_index < len(ids):
            v = ids[gpu_index]
            self.h = pynvml.nvmlDeviceGetHandleByIndex(int(v)) if v.isdigit() else pynvml.nvmlDeviceGetHandleByUUID(v)
        else:
            self.h = pynvml.nvmlDeviceGetHandleByIndex(gpu_index)
        self.rows, self.run, self.th = [], False, None
        nv = pynvml
        self.bits = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else 0x8,
                     "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
        self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))

    def _loop(self):
        nv = self.nv
        while self.run:
            try:
                sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                pw = nv.nvmlDeviceGetPowerUsage(self.h) * 1e-3
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.rows.append((time.time(), sm, self.smax, pw, {k for k, b in self.bits.items() if mask & b}))
            except Exception:
                pass
            time.sleep(0.05)

    def start(self):
        self.run = True
        self.th = threading.Thread(target=self._loop, daemon=True)
        self.th.start()

    def wait_first(self, timeout: float = 5.0):
        t = time.time()
        while not self.rows and time.time() - t < timeout:
            time.sleep(0.02)

    def stop(self, t0: float, t1: float) -> dict:
        time.sleep(0.06)
        self.run = False
        if self.th is not None:
            self.th.join(timeout=2)
        return _clock_summary(self.rows, t0, t1, "nvml")


class NoSampler:
    def __init__(self, why: str = "clock sampling disabled"):
        self.why = why

    def start(self):
        pass

    def wait_first(self, timeout: float = 0.0):
        pass

    def stop(self, t0: float, t1: float) -> dict:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [self.why], "samples": 0, "source": "none"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md, clocks line); the fallback when
    NVML cannot be imported (--clock-sampler nvidia-smi forces it)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.idx = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.strip().split(",")]
            try:
                self.rows.append((time.time(), float(f[1]), float(f[2]), float(f[3]),
                                  {nm for nm, v in zip(CLOCK_REASONS, f[4:8]) if v.lower().startswith("active")}))
            except (ValueError, IndexError):
                continue

    def wait_first(self, timeout: float = 5.0):
        t = time.time()
        while self.proc is not None and not self.rows and time.time() - t < timeout:
            time.sleep(0.02)

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "source": "nvidia-smi"}
        time.sleep(0.15)
        self.proc.terminate()
        try:  # nvidia-smi's exit briefly stalls the driver: be sure it is gone before anything else is timed
            self.proc.wait(timeout=10)
        except Exception:
            self.proc.kill()
        time.sleep(0.5)
        return _clock_summary(self.rows, t0, t1, "nvidia-smi")


def make_clock_sampler(kind: str, gpu_index: int):
    if kind == "none":
        return NoSampler()
    if kind == "nvml":
        try:
            return NvmlSampler(gpu_index)
        except Exception:
            pass  # no pynvml / no NVML on this box: the nvidia-smi process
    return ClockSampler(gpu_index)


# ------------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_step(s) -> float:
    """One pass of the whole path by the oracle (graph, halos, gather, SP2, scatter); returns seconds."""
    import oracle as o
    t0 = time.perf_counter()
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    dt = time.perf_counter() - t0
    assert r.iters_done == s.iters
    return dt


def cpu_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def sample_description(s, workload_mol: int) -> str:
    if s.meta["n_mol"] == workload_mol:
        return (f"the whole workload: {s.meta['n_mol']}-molecule water box ({s.n} orbitals, {s.n_part} communities), "
                f"tau={s.tau:g}, {s.iters} SP2 iterations, one full pass of the oracle per step")
    return (f"{s.meta['n_mol']}-molecule water box ({s.n} orbitals, {s.n_part} communities): same construction, density, "
            f"tau={s.tau:g} and {s.iters} SP2 iterations as the workload; the path is linear scaling, so cost per orbital "
            "does not depend on the box size")


def oracle_sample_molecules(workload: str, oracle_passes: int, budget_s: float) -> int:
    """The largest box (the workload itself if it fits) whose `oracle_passes` oracle passes end within budget_s on the
    cores this process may use; the oracle's cost is linear in the number of molecules (same density, same tau)."""
    full = WORKLOADS[workload][0] or 4096
    per_mol = ORACLE_S_PER_MOLECULE_16_CORES * max(1.0, 16.0 / cpu_cores())
    n_mol = full
    while n_mol > 256 and oracle_passes * n_mol * per_mol > budget_s:
        n_mol //= 2
    return n_mol


def run_reference(args) -> None:
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    total = args.steps + args.warmup
    # the real workload when all passes fit ~5 minutes (28 s per pass on 16 cores), else a smaller box of the same model
    n_mol = oracle_sample_molecules(args.workload, total, 300.0)
    import gbe_inputs as gi
    s = gi.water_box(n_mol, n_mol // 8, seed=0)
    for _ in range(args.warmup):
        oracle_step(s)
    times = [oracle_step(s) for _ in range(args.steps)]
    dt = float(np.mean(times))
    v = s.n / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "note": "CPU oracle (numpy/scipy, host BLAS), bounded sample per step",
                   "sample_is_the_workload": s.meta["n_mol"] == (WORKLOADS[args.workload][0] or -1)},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cpu_cores(), "kind": "oracle",
                         "sample": sample_description(s, WORKLOADS[args.workload][0] or -1)},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# N > 1: replicas only - the single cross-rank step is the reduction of the timings
# ------------------------------------------------------------------------------------------------
def over_ranks(x: float, op: str, device: str) -> float:
    """max / sum of a per-rank scalar over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_all_ranks: float, steps: int, ms_max_over_ranks: float) -> float:
    """Whole-job throughput: units processed by ALL ranks per step x steps / the slowest rank's time."""
    return units_all_ranks * steps / (ms_max_over_ranks * 1e-3)


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
def pinned_host_csr(H):
    """The CSR arrays of H in pinned host memory (numpy views of pinned torch tensors)."""
    import torch
    import gbe_inputs as gi
    keep = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (H.row_ptr, H.col_idx, H.val)]
    h = gi.CSR(H.n, keep[0].numpy(), keep[1].numpy(), keep[2].numpy())
    h._keep = keep
    return h


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_1603_00937_b200 import build as gbe_build
    if rank == 0:
        gbe_build.build()
    if world > 1:
        dist.barrier()
    import paper_1603_00937_b200 as gbe
    gbe.lib()

    sm_count = torch.cuda.get_device_properties(local).multi_processor_count

    s = make_system(args.workload, seed=rank)  # replicas: one independent seeded box per rank
    stream = torch.cuda.current_stream()
    Hd = gbe.DeviceCSR.from_host(s.H)
    Hh = pinned_host_csr(s.H)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    # sizes are fixed by the graph: build once to allocate outputs/workspace outside the timed region
    part_t = None if s.meta.get("kind") == "water" else torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    part_h = None if part_t is None else np.asarray(s.part, dtype=np.int32)
    g0 = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    info = dict(g0.info)
    ws = g0.new_workspace()
    D_val = torch.empty(info["nnz_D"], dtype=torch.float64, device="cuda")
    D_host = torch.empty(info["nnz_D"], dtype=torch.float64).pin_memory()
    g0.free()

    def step_device():
        g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part, stream=stream)
        gbe.gbe_density(Hd, g, s.n_occ, s.iters, -1.0, workspace=ws, D_val=D_val, want_log=False, stream=stream)
        g.free()  # inside the step: the graph of a step is released when its D is done (returns its arrays to the pool)

    def step_host():
        g = gbe.gbe_build_graph_host(Hh, s.tau, part_h, s.n_part, stream=stream)
        # H_host=None: the device copy uploaded by gbe_build_graph_host is reused (one upload per step)
        gbe.gbe_density_host(None, g, s.n_occ, s.iters, -1.0, workspace=ws, D_val_host=D_host.numpy(), stream=stream)
        g.free()

    step_ms_log = []

    def timed_region(step, steps):
        """K steps, each bracketed by CUDA events on the launching stream, L2 flushed (untimed) between steps."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        n0 = gbe.gbe_launch_count()
        for e0, e1 in ev:
            flush.zero_()
            e0.record(stream)
            step()
            e1.record(stream)
        torch.cuda.synchronize()
        launches = gbe.gbe_launch_count() - n0
        if world > 1:
            dist.barrier()
        ms = [e0.elapsed_time(e1) for e0, e1 in ev]
        step_ms_log.append([round(x, 3) for x in ms])
        return float(np.sum(ms)), int(launches)

    # the sampler runs from before the warm-up: whatever attaching it costs is paid outside the timed region
    clocks = make_clock_sampler(args.clock_sampler, local)
    clocks.start()
    for _ in range(max(args.warmup, 3)):
        step_device()
    torch.cuda.synchronize()
    clocks.wait_first()
    t_wall0 = time.time()
    total_ms, launches = timed_region(step_device, args.steps)
    t_wall1 = time.time()
    clk = clocks.stop(t_wall0, t_wall1)

    # end to end: HOST buffers through the C ABI, copies inside the timed region
    for _ in range(max(args.warmup, 3)):
        step_host()
    e2e_ms, _ = timed_region(step_host, args.steps)

    # roofline denominator: cuBLAS DGEMM in this process, AFTER the timed regions (its 4 s of back-to-back GEMMs heat
    # the part and its 1.5 GB of torch allocations disturb the pool; neither belongs in front of the steps)
    fp64_peak = measure_fp64_peak(torch)

    # per-kernel device times, same process, same inputs (CUDA events around every launch of gbe_density)
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    ph = None
    for _ in range(2):
        flush.zero_()
        _, ph = gbe.gbe_density_timed(Hd, g, s.n_occ, s.iters, -1.0, workspace=ws, D_val=D_val)
    # graph build alone
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part).free()
    e1.record(stream)
    torch.cuda.synchronize()
    graph_ms = e0.elapsed_time(e1)

    total_ms_max, e2e_ms_max = over_ranks(total_ms, "max", "cuda"), over_ranks(e2e_ms, "max", "cuda")
    orbitals_all = over_ranks(float(s.n), "sum", "cuda")
    value = job_throughput(orbitals_all, args.steps, total_ms_max)
    e2e_value = job_throughput(orbitals_all, args.steps, e2e_ms_max)

    if rank == 0:
        peaks = load_peaks()
        x2_ms = ph["x2_ms"] / max(1, ph["x2_launches"])
        per_s = 1.0 / (x2_ms * 1e-3) * 1e-12
        sym_tf = info["sp2_sym_flops_per_iter"] * per_s    # what the method needs with X = X^T ("m^3 if symmetry is exploited")
        alg_tf = info["sp2_flops_per_iter"] * per_s        # 2 m^3, symmetry not counted: an EFFECTIVE rate, never divided by a peak
        exec_tf = info["sp2_exec_flops_per_iter"] * per_s  # issued to the FP64 tensor pipe (8x8 sub-tiles on/above the diagonal, K padded to ld)
        peak_tf = fp64_peak["sustained_tflops"]            # the X^2 launches run back to back inside a long step
        issue_tf = (DMMA_FLOP_PER_CLK_PER_SM * sm_count * clk["sm_mhz"] * 1e6 * 1e-12) if clk.get("sm_mhz") else None
        traffic, traffic_note = x2_traffic(args.workload)
        nnzH = int(s.H.nnz)
        gather_bytes = info["dense_elems"] * 8 + 12.0 * nnzH * info["sum_m"] / info["n"]   # every H row re-read by each subgraph holding it
        gather_dram_bytes = info["dense_elems"] * 8 + 12.0 * nnzH + 8.0 * (info["n"] + 1)  # compulsory: write X once, read H once
        scatter_bytes = 16.0 * info["nnz_D"]
        gather_gbs = gather_bytes / (ph["gather_ms"] * 1e-3) * 1e-9
        gather_dram_gbs = gather_dram_bytes / (ph["gather_ms"] * 1e-3) * 1e-9
        scatter_gbs = scatter_bytes / (ph["scatter_ms"] * 1e-3) * 1e-9
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {
                "workload": f"{args.workload}: {s.meta['kind']}, {s.n} orbitals, "
                            f"n_occ={s.n_occ:g}, tau={s.tau:g}, {s.n_part} communities, {s.iters} SP2 iterations, FP64",
                "step": "gbe_build_graph + gbe_density (rows 0-6)", "parallelism": "replicas only" if world > 1 else "1 GPU",
                "l2": "256 MiB buffer written between timed steps; dense batch (2 x %.2f GB) exceeds L2" % (info["dense_elems"] * 8e-9),
                "m_mean": info["sum_m"] / info["n_part"], "m_max": info["max_m"], "nnz_H": nnzH, "nnz_D": info["nnz_D"],
            },
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms_max / args.steps,
                    "h2d_bytes_per_step": int(s.H.row_ptr.nbytes + s.H.col_idx.nbytes + s.H.val.nbytes),
                    "d2h_bytes_per_step": int(info["nnz_D"] * 8)},
            "gpu_launches": launches,
            "ms_steps": {"device": step_ms_log[0], "e2e": step_ms_log[-1]},
            "clocks": clk,
            "roofline": {
                "kernel": "k_x2_tma (Y = X X^T on DMMA.8x8x4, panels by 2-D TMA, fused branch/trace epilogue)", "bound": "tensor",
                "achieved": sym_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": sym_tf / peak_tf,
                "traffic": traffic, "traffic_note": traffic_note,
                "algorithmic_bytes_per_launch": 16.0 * info["dense_elems"],
                "basis": "sum_p m_p^2 (m_p + 1) flop per launch - one SP2 iteration of the whole batch with X = X^T used "
                         "(entries on or above the diagonal of X_p^2, unpadded; gbe_graph_info.sp2_sym_flops_per_iter) - / mean "
                         "CUDA-event time of the %d full launches" % ph["x2_launches"],
                "flop_per_launch": info["sp2_sym_flops_per_iter"], "ms_per_launch": x2_ms,
                "peak_source": "cuBLAS DGEMM f64 8192^3 (torch.matmul), this run, sustained over %d back-to-back calls; "
                               "MEASURED_PEAKS.json has no FP64 entry" % fp64_peak["reps_sustained"],
                "peak_burst": fp64_peak["burst_tflops"],
                "issue_rate_peak": issue_tf,
                "issue_rate_source": "%g flop/clk/SM (DMMA.8x8x4 every 16 cycles per SM sub-partition, profiles/"
                                     "r01_fp64_peak_probe.md) x %d SMs x median SM clock sampled in the timed region"
                                     % (DMMA_FLOP_PER_CLK_PER_SM, sm_count),
                "frac_of_issue_rate": sym_tf / issue_tf if issue_tf else None,
                "executed_tflops": exec_tf, "executed_frac_of_issue_rate": exec_tf / issue_tf if issue_tf else None,
                "effective_tflops_2m3": alg_tf,
                "last_iteration": {"note": "launch %d of %d computes the tiles with a core row only (Eq.(6): the core "
                                           "columns are kept); timed apart and not part of the mean above"
                                           % (s.iters, s.iters),
                                   "ms": ph["x2_last_ms"], "tiles": info["n_tiles_last"], "tiles_full": info["n_tiles"],
                                   "executed_tflops": info["sp2_exec_flops_last_iter"] / max(ph["x2_last_ms"], 1e-6) * 1e-9},
            },
            "phases_ms": {"graph_build": graph_ms, "bounds": ph["bounds_ms"], "gather": ph["gather_ms"],
                          "x2": ph["x2_ms"] + ph["x2_last_ms"],
                          "trace_branch": ph["trace_ms"], "scatter": ph["scatter_ms"], "density_total": ph["total_ms"]},
            "sp2_solves_per_s": info["n_part"] / ((ph["x2_ms"] + ph["x2_last_ms"] + ph["trace_ms"]) * 1e-3),
            "hbm": {"peak_gbs": peaks["hbm_gbs"], "peak_source": peaks["source"], "nominal_gbs": HBM_NOMINAL_GBS,
                    "gather_gbs": gather_gbs, "gather_frac": gather_gbs / peaks["hbm_gbs"],
                    "gather_frac_nominal": gather_gbs / HBM_NOMINAL_GBS,
                    "gather_dram_gbs": gather_dram_gbs, "gather_dram_frac": gather_dram_gbs / peaks["hbm_gbs"],
                    "gather_note": "gather_gbs counts SURVEY 8(a)'s bytes (each H row read by every subgraph that holds "
                                   "it; those re-reads are L2 hits); gather_dram_gbs counts compulsory DRAM bytes only "
                                   "(X written once, H read once)",
                    "scatter_gbs": scatter_gbs, "scatter_frac": scatter_gbs / peaks["hbm_gbs"],
                    "scatter_frac_nominal": scatter_gbs / HBM_NOMINAL_GBS},
        }
        if world == 1 and not args.no_cpu_baseline:
            import gbe_inputs as gi
            # one pass of the oracle over the workload itself when that is ~30 s of CPU work (the 4,096-molecule box on
            # 16 cores), else over the largest smaller box of the same model that is
            full_mol = WORKLOADS[args.workload][0] or -1
            n_mol = oracle_sample_molecules(args.workload, 1, 45.0)
            cs = s if (n_mol == full_mol and s.meta.get("kind") == "water") else gi.water_box(n_mol, n_mol // 8, seed=0)
            dt = oracle_step(cs)
            line["cpu_baseline"] = {"value": cs.n / dt, "unit": UNIT, "cores": cpu_cores(), "kind": "oracle",
                                    "seconds": dt, "sample": sample_description(cs, full_mol)}
        print(json.dumps(line), flush=True)
    g.free()
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs[4]: threshold x partition sweep on the 24,576-orbital water box
# ------------------------------------------------------------------------------------------------
def run_sweep(args) -> None:
    """tau in {1e-3..1e-7} x communities in {128,256,512,1024} on one geometry: halo size distribution, cost
    (sum 2 m^3, the paper's cost law P:L78), throughput, and the error against the exact zero-temperature projector.
    The exact projector comes from torch.linalg.eigh on the GPU (a library call, used for this report only).
    One JSON line per point; `--sweep-out FILE` also writes a markdown table."""
    import torch
    import gbe_inputs as gi
    from paper_1603_00937_b200 import build as gbe_build
    gbe_build.build()
    import paper_1603_00937_b200 as gbe

    n_mol = WORKLOADS[args.workload][0]
    taus = [float(x) for x in args.sweep_taus.split(",")] if args.sweep_taus else [1e-3, 1e-4, 1e-5, 1e-6, 1e-7]
    parts = [n_mol // 32, n_mol // 16, n_mol // 8, n_mol // 4]
    # --gapped: the variant of the water model with a HOMO-LUMO gap (oxygens >= 2.4 A apart, 3 electrons per molecule,
    # reading A-15), run to idempotency: there the error against the exact projector measures the method, not the model
    wkw = dict(min_oo=2.4, occ_per_mol=3.0) if args.gapped else {}
    idem_tol = 1e-10 if args.gapped else -1.0
    base = gi.water_box(n_mol, parts[2], seed=0, **wkw)
    Hd = gbe.DeviceCSR.from_host(base.H)
    n, n_occ = base.n, base.n_occ
    Dex = None
    if not args.no_exact:
        t0 = time.time()
        Hdense = torch.from_numpy(base.H.to_dense()).cuda()
        w, V = torch.linalg.eigh(Hdense)
        del Hdense
        k = int(round(n_occ))
        gap = float(w[k] - w[k - 1])
        eband_exact = float(w[:k].sum())  # Tr[D_exact H] = sum of the occupied eigenvalues
        Dex = V[:, :k] @ V[:, :k].T
        del V
        torch.cuda.synchronize()
        sys.stderr.write(f"exact projector: {time.time() - t0:.1f} s, HOMO-LUMO gap {gap:.3e} eV\n")
    rows = []
    for tau in taus:
        for n_part in parts:
            torch.cuda.synchronize()
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            gbe.gbe_build_graph(Hd, tau, None, n_part).free()  # warm-up of the allocator for this size
            e0.record()
            g = gbe.gbe_build_graph(Hd, tau, None, n_part)
            e1.record()
            if args.sp2_path:
                gbe.gbe_graph_set_sp2_path(g, args.sp2_path)
            info = g.info
            ws = g.new_workspace()
            D_val = torch.empty(info["nnz_D"], dtype=torch.float64, device="cuda")
            gbe.gbe_density(Hd, g, n_occ, base.iters, idem_tol, workspace=ws, D_val=D_val, want_log=False)  # warm-up
            torch.cuda.synchronize()
            e1.record()
            _, log = gbe.gbe_density(Hd, g, n_occ, base.iters, idem_tol, workspace=ws, D_val=D_val, want_log=True)
            e2.record()
            torch.cuda.synchronize()
            _, ph = gbe.gbe_density_timed(Hd, g, n_occ, base.iters, idem_tol, workspace=ws, D_val=D_val)
            # the paper's own mode: the sequence just logged, given beforehand, no trace reduction between products
            seq = log.branch
            gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=ws, D_val=D_val, want_log=False)
            torch.cuda.synchronize()
            e3, e4 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e3.record()
            gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=ws, D_val=D_val, want_log=False)
            e4.record()
            torch.cuda.synchronize()
            preset_ms = e3.elapsed_time(e4)
            ex = g.export()
            m = (ex["sub_ptr"][1:] - ex["sub_ptr"][:-1]).double()
            rec = {"sweep": args.workload, "tau": tau, "n_part": n_part, "m_min": int(m.min()), "m_mean": float(m.mean()),
                   "m_max": int(m.max()), "sum_2m3": info["sp2_flops_per_iter"], "nnz_S": info["nnz_S"],
                   "nnz_D": info["nnz_D"], "density_ms": e1.elapsed_time(e2),
                   "orbitals_per_s": n / (e1.elapsed_time(e2) * 1e-3),
                   "sp2_loop_ms": ph["x2_ms"] + ph["x2_last_ms"] + ph["trace_ms"], "gather_ms": ph["gather_ms"],
                   "scatter_ms": ph["scatter_ms"],
                   "sp2_exec_tflops": info["sp2_exec_flops_per_iter"] * max(0, log.iters_done - 1) / max(1e-9, ph["x2_ms"] * 1e-3) * 1e-12,
                   "preset_no_trace_ms": preset_ms, "x2_tma": int(info["x2_tma"]), "iters_done": int(log.iters_done), "sp2_path": int(info["sp2_path_chosen"]),
                   "n_small": int(info["n_small"]), "n_bins": int(info["n_bins"]),
                   "sp2_tflops_alg": (info["sp2_flops_per_iter"] * max(0, log.iters_done - 1) + info["sp2_flops_last_iter"])
                                     / (e1.elapsed_time(e2) * 1e-3) * 1e-12,
                   "trace_minus_nocc": float(log.t1[-1] - n_occ), "idempotency_residual": float(log.t1[-1] - log.t2[-1])}
            if Dex is not None:
                mx, f_in, f_all = gbe.gbe_error_norms(g, D_val, Dex)  # Fig.2
                rec["max_abs_err_vs_exact"] = mx
                rec["frobenius_err_per_orbital"] = float(np.sqrt(f_in)) / n          # over the stored entries of D
                rec["frobenius_err_full_per_orbital"] = float(np.sqrt(f_all)) / n    # D = 0 where it stores nothing
                # band energy E_band = Tr[D H] (Fig.2 P:L199 plots its error per atom)
                rec["eband_err_per_orbital"] = (gbe.gbe_expectation(g, D_val, Hd) - eband_exact) / n
            rows.append(rec)
            print(json.dumps(rec), flush=True)
            g.free()
            del ws, D_val, ex
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            f.write("| tau | communities | m min/mean/max | sum 2m^3 per iteration | SP2 iterations | density ms | orbitals/s | TFLOP/s (2m^3) | "
                    "max abs err vs exact | Frobenius err / orbital (stored entries) | Frobenius err / orbital (full matrix) | E_band err / orbital (eV) | Tr D - n_occ |\n|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write(f"| {r['tau']:g} | {r['n_part']} | {r['m_min']}/{r['m_mean']:.0f}/{r['m_max']} | {r['sum_2m3']:.3g} | "
                        f"{r['iters_done']} | {r['density_ms']:.1f} | {r['orbitals_per_s']:.3g} | {r['sp2_tflops_alg']:.1f} | "
                        f"{r.get('max_abs_err_vs_exact', float('nan')):.3g} | {r.get('frobenius_err_per_orbital', float('nan')):.3g} | "
                        f"{r.get('frobenius_err_full_per_orbital', float('nan')):.3g} | "
                        f"{r.get('eband_err_per_orbital', float('nan')):.3g} | "
                        f"{r['trace_minus_nocc']:.3g} |\n")


def run_fermi(args) -> None:
    """the finite-temperature Chebyshev expansion (Eq.(7)) on the bench workload, one JSON line."""
    import torch
    from paper_1603_00937_b200 import build as gbe_build
    gbe_build.build()
    import paper_1603_00937_b200 as gbe
    s = make_system(args.workload, 0)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    info = g.info
    ws = torch.empty(info["workspace_bytes_fermi"], dtype=torch.uint8, device="cuda")
    D_val = torch.empty(info["nnz_D"], dtype=torch.float64, device="cuda")
    order, mu, beta = args.fermi_order, -11.0, 0.8
    gbe.gbe_density_fermi(Hd, g, mu, beta, order, workspace=ws, D_val=D_val)
    ms = []
    for _ in range(max(1, args.steps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _, ne = gbe.gbe_density_fermi(Hd, g, mu, beta, order, workspace=ws, D_val=D_val, want_n_elec=False)
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    t = float(np.median(ms))
    print(json.dumps({"fermi": args.workload, "order": order, "mu": mu, "beta": beta, "ms": t,
                      "ms_per_term": t / (order - 1), "orbitals_per_s": s.n / (t * 1e-3),
                      "tflops_alg": info["sp2_flops_per_iter"] * (order - 1) / (t * 1e-3) * 1e-12}), flush=True)


def run_timeline(args) -> None:
    """Timeline INSIDE the two hot kernels from %globaltimer stamps (profiles/r02_small_m_ncu.md, r02_x2_timeline.md).
    Runs on the instrumented copy of the library (python -m paper_1603_00937_b200.build --stamps -> libgbe_stamps.so; the
    stamps are compiled out of libgbe.so and add ~10 % to a packed launch), so nothing printed here is a bench value.
      packed: the 1,024-community point of the sweep (water box, tau = 1e-3): per bin of k_sp2_packed, means over the bins
              of one launch in the middle of the loop, split by wave;
      x2:     the bench workload: per CTA of k_x2_tma for two consecutive launches - tile durations, how many CTAs run
              near the end of a launch (the tail), and the hand-over to the next launch."""
    import ctypes as C
    import torch
    import gbe_inputs as gi
    from paper_1603_00937_b200 import build as gbe_build
    import paper_1603_00937_b200.binding as binding
    binding.LIB_PATH = gbe_build.build(stamps=True)
    import paper_1603_00937_b200 as gbe
    l = binding.lib()
    if args.timeline == "packed":
        s = gi.water_box(4096, 1024, seed=0, tau=1e-3)
    else:
        s = make_system(args.workload, seed=0)
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = None if s.meta.get("kind") == "water" else torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    info = g.info
    ws = g.new_workspace()
    D = torch.empty(info["nnz_D"], dtype=torch.float64, device="cuda")
    for _ in range(3):  # the stamps of the last call stay
        gbe.gbe_density(Hd, g, s.n_occ, 40, -1.0, workspace=ws, D_val=D, want_log=False)
    torch.cuda.synchronize()
    us = 1e-3
    out = {"timeline": args.timeline, "n": s.n, "n_part": s.n_part, "sp2_path": info["sp2_path_chosen"], "unit": "us"}
    if args.timeline == "packed":
        if info["sp2_path_chosen"] != 3:
            raise SystemExit("--timeline packed: the library did not choose the packed kernel for this system")
        I, B, W = C.c_int(), C.c_int(), C.c_int()
        l.gbe_stamps_packed_shape(C.byref(I), C.byref(B), C.byref(W))
        I, B, W = I.value, B.value, W.value
        buf = np.zeros(I * B * W, dtype=np.uint64)
        l.gbe_stamps_packed.argtypes = [C.c_void_p, C.c_size_t]
        rc = l.gbe_stamps_packed(buf.ctypes.data, buf.nbytes)
        if rc != 0:
            raise SystemExit(f"gbe_stamps_packed: {rc}")
        nb = info["n_bins"]
        st = buf.reshape(I, B, W)[:, :nb, :].astype(np.float64)
        out["bins"] = nb
        out["launches"] = []
        for it in (10, 20, 30):
            a = st[it]
            prev_end = st[it - 1][:, 5].max()
            row = {"iter": it, "launch_to_launch": round((a[:, 5].max() - prev_end) * us, 2),
                   "first_entry_rel_prev_end": round((a[:, 0].min() - prev_end) * us, 2),
                   "release_rel_prev_end": [round((a[:, 2].min() - prev_end) * us, 2), round((a[:, 2].max() - prev_end) * us, 2)],
                   "waves": []}
            order = np.argsort(a[:, 0])
            for idx in (order[:148], order[148:]):
                if len(idx) == 0:
                    continue
                e = a[idx]
                done = e[:, 8:40].max(axis=1)
                land = (e[:, 40:56] - e[:, 2:3]) * us
                land[e[:, 40:56] == 0] = np.nan
                row["waves"].append({
                    "bins": int(len(idx)),
                    "setup": round((e[:, 1] - e[:, 0]).mean() * us, 2),
                    "wait": round((e[:, 2] - e[:, 1]).mean() * us, 2),
                    "copies_issued": round((e[:, 3] - e[:, 2]).mean() * us, 2),
                    "step5": round((e[:, 7] - e[:, 3]).mean() * us, 2),
                    "slot0_landed_after_release": round(float(np.nanmean(land[:, 0])), 2),
                    "last_slot_landed_after_release": round(float(np.nanmean(np.nanmax(land, axis=1))), 2),
                    "first_unit_after_step5": round((e[:, 4] - e[:, 7]).mean() * us, 2),
                    "units": [round((done - e[:, 4]).mean() * us, 2), round((done - e[:, 4]).max() * us, 2)],
                    "pair_published_after_units": round((e[:, 5] - done).mean() * us, 2),
                    "bin_total": [round((e[:, 5] - e[:, 0]).mean() * us, 2), round((e[:, 5] - e[:, 0]).max() * us, 2)],
                })
            out["launches"].append(row)
    else:
        I0, I, B, W = C.c_int(), C.c_int(), C.c_int(), C.c_int()
        l.gbe_stamps_x2_shape(C.byref(I0), C.byref(I), C.byref(B), C.byref(W))
        I0, I, B, W = I0.value, I.value, B.value, W.value
        buf = np.zeros(I * B * W, dtype=np.uint64)
        l.gbe_stamps_x2.argtypes = [C.c_void_p, C.c_size_t]
        rc = l.gbe_stamps_x2(buf.ctypes.data, buf.nbytes)
        if rc != 0:
            raise SystemExit(f"gbe_stamps_x2: {rc}")
        nt = info["n_tiles"]
        if nt > B:
            raise SystemExit(f"--timeline x2: {nt} tiles, the stamp array holds {B}")
        st = buf.reshape(I, B, W)[:, :nt, :].astype(np.float64)
        if not st[:, :, 0].all():
            raise SystemExit("--timeline x2: k_x2_tma did not run these launches (not the TMA kernel on this system?)")
        out["tiles"] = nt
        out["launches"] = []
        slots = 4 * torch.cuda.get_device_properties(0).multi_processor_count
        for k in range(I):
            a = st[k]
            t0, t_end = a[:, 0].min(), a[:, 2].max()
            dur, ml, ep = a[:, 2] - a[:, 0], a[:, 1] - a[:, 0], a[:, 2] - a[:, 1]
            sm = a[:, 3].astype(int)
            last_end = np.array([a[sm == j, 2].max() for j in np.unique(sm)])
            out["launches"].append({
                "iter": I0 + k, "span": round((t_end - t0) * us, 1),
                "tile_mean": round(dur.mean() * us, 2), "main_loop_mean": round(ml.mean() * us, 2), "epilogue_mean": round(ep.mean() * us, 2),
                "sum_tile_time_over_slots": round(dur.sum() / slots * us, 1), "slots": slots,
                "sm_idle_before_end_mean": round((t_end - last_end).mean() * us, 1), "sm_idle_before_end_max": round((t_end - last_end).max() * us, 1),
                "running_ctas_before_end": {str(b): int(((a[:, 0] <= t_end - b * 1e3) & (a[:, 2] > t_end - b * 1e3)).sum())
                                            for b in (100, 60, 40, 20, 10, 5)},
            })
        if I >= 2:
            out["handover"] = {"end_to_first_cta_of_next": round((st[1][:, 0].min() - st[0][:, 2].max()) * us, 2),
                               "end_to_first_epilogue_of_next": round((st[1][:, 1].min() - st[0][:, 2].max()) * us, 1)}
    print(json.dumps(out), flush=True)


def run_md(args) -> None:
    """The paper's use of the method, one quantum-MD step at a time, on the bench workload: S(t) from Eq.(8)
    with D(t - dt) and the moved Hamiltonian H(t) (gbe_update_graph), the density with the SP2 sequence of the previous
    step (gbe_density_preset, no trace reduction between the products), the band energy Tr[D H] (gbe_expectation).
    H(t) = the seeded box with every element moved by up to 0.1 % per step, kept symmetric (a stand-in for moving atoms:
    same pattern, changing values).  Step 0 is an ordinary build + trace-driven density.  One JSON line per step."""
    import torch
    from paper_1603_00937_b200 import build as gbe_build
    gbe_build.build()
    import paper_1603_00937_b200 as gbe
    import gbe_inputs as gi
    # the gapped variant of the water model (oxygens >= 2.4 A apart, 3 electrons per molecule, reading A-15): D decays
    # exponentially there, as in the paper's systems; on the gapless default box |D_ij| >= tau reaches across the box and
    # Eq.(8)'s paths of length two make every community the whole system
    n_mol = WORKLOADS[args.workload][0]
    s = gi.water_box(n_mol, n_mol // 8, seed=0, min_oo=2.4, occ_per_mol=3.0) if n_mol else make_system(args.workload, seed=0)
    tau_d = args.md_tau
    Hs = s.H.to_scipy().tocsr()
    part_t = None if s.meta.get("kind") == "water" else torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()

    def moved(step):
        m = Hs.copy()
        m.data = m.data * (1.0 + 1e-3 * np.cos(np.arange(m.nnz) * 0.37 + step))
        return gbe.DeviceCSR.from_host(gi.CSR.from_scipy((m + m.T) * 0.5))

    ev = lambda: torch.cuda.Event(enable_timing=True)
    Hd = moved(0)
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    D, log = gbe.gbe_density(Hd, g, s.n_occ, s.iters, -1.0)
    seq = log.branch
    for step in range(1, args.steps + 1):
        Hd = moved(step)
        torch.cuda.synchronize()
        e = [ev() for _ in range(4)]
        e[0].record()
        g1 = gbe.gbe_update_graph(g, D, Hd, tau_d, part_t, s.n_part)
        e[1].record()
        info = g1.info
        if info["workspace_bytes"] > 100e9:
            print(json.dumps({"md_step": step, "error": "Eq.(8) graph too dense for this tau", "tau_graph": tau_d,
                              "m_mean": info["sum_m"] / info["n_part"], "m_max": info["max_m"],
                              "workspace_gb": info["workspace_bytes"] * 1e-9}), flush=True)
            return
        ws = g1.new_workspace()
        D1 = torch.empty(info["nnz_D"], dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        e[1].record()
        gbe.gbe_density_preset(Hd, g1, seq, trace_every_iteration=False, workspace=ws, D_val=D1, want_log=False)
        e[2].record()
        eband = gbe.gbe_expectation(g1, D1, Hd)
        e[3].record()
        torch.cuda.synchronize()
        # the sequence for the next step: the one a trace-driven run of THIS step chooses (untimed; an MD code would
        # keep the sequence while the gap estimate holds)
        _, lg = gbe.gbe_density(Hd, g1, s.n_occ, s.iters, -1.0, workspace=ws, D_val=torch.empty_like(D1))
        same = bool(np.array_equal(lg.branch, seq))
        seq = lg.branch
        print(json.dumps({"md_step": step, "workload": args.workload, "n": s.n, "n_part": s.n_part, "tau_graph": tau_d,
                          "nnz_S": info["nnz_S"], "m_mean": info["sum_m"] / info["n_part"], "m_max": info["max_m"],
                          "nnz_D": info["nnz_D"], "sp2_path": info["sp2_path_chosen"],
                          "graph_update_ms": e[0].elapsed_time(e[1]), "density_preset_ms": e[1].elapsed_time(e[2]),
                          "expectation_ms": e[2].elapsed_time(e[3]),
                          "step_ms": e[0].elapsed_time(e[1]) + e[1].elapsed_time(e[3]),
                          "orbitals_per_s": s.n / ((e[0].elapsed_time(e[1]) + e[1].elapsed_time(e[3])) * 1e-3),
                          "band_energy": eband, "sequence_unchanged": same}), flush=True)
        g.free()
        g, D = g1, D1
    g.free()


def run_trace_build(args) -> None:
    """Timeline of gbe_build_graph (steps 0-2) on the bench workload: every kernel, copy and memset with its start time
    (CUPTI through torch.profiler - a library used for this report only), so that device IDLE time shows: the span of one
    build, the time the device is busy in it, and the gaps.  One JSON line; profiles/r02_graph_build.md records it."""
    import re
    import torch
    from torch.profiler import profile, ProfilerActivity
    from paper_1603_00937_b200 import build as gbe_build
    gbe_build.build()
    import paper_1603_00937_b200 as gbe
    s = make_system(args.workload, seed=0)
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = None if s.meta.get("kind") == "water" else torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    for _ in range(3):
        gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part).free()
    torch.cuda.synchronize()
    with profile(activities=[ProfilerActivity.CPU, ProfilerActivity.CUDA]) as prof:
        for _ in range(3):
            gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part).free()
        torch.cuda.synchronize()
    import tempfile
    with tempfile.TemporaryDirectory() as td:  # the chrome-trace export is the profiler's stable interface
        fn = os.path.join(td, "trace.json")
        prof.export_chrome_trace(fn)
        with open(fn) as f:
            tr = json.load(f)["traceEvents"]
    ev = sorted((e["ts"], e["ts"] + e["dur"], e["name"]) for e in tr if e.get("cat") in ("kernel", "gpu_memcpy", "gpu_memset"))
    starts = [i for i, e in enumerate(ev) if "k_row_bounds" in e[2]]
    seg = ev[starts[1]:starts[2]]  # the second of the three profiled builds
    t0, t1 = seg[0][0], max(e[1] for e in seg)
    busy = sum(e[1] - e[0] for e in seg)
    gaps, prev = [], None
    for a, b, name in seg:
        m = re.search(r"(k_[a-z0-9_]+(<[^>]*>)?)", name)
        if prev is not None and a - prev > 8.0:
            gaps.append({"at_us": round(a - t0, 1), "gap_us": round(a - prev, 1), "before": m.group(1) if m else name[:40]})
        prev = max(prev or 0, b)
    top = sorted(({"name": (re.search(r"(k_[a-z0-9_]+(<[^>]*>)?)", n) or re.match(r".{0,40}", n)).group(0), "us": round(b - a, 1)}
                  for a, b, n in seg), key=lambda d: -d["us"])[:8]
    print(json.dumps({"trace_build": args.workload, "n": s.n, "n_part": s.n_part, "device_ops": len(seg),
                      "span_us": round(t1 - t0, 1), "busy_us": round(busy, 1), "idle_us": round(t1 - t0 - busy, 1),
                      "gaps_over_8us": gaps, "longest": top}), flush=True)


def run_waves(args) -> None:
    """SURVEY 8(f) item 1 in a bounded workspace: gbe_density_preset without traces on the whole batch against the same call
    in a workspace of --waves-gb GB (waves of communities: no exchange between the expansions).  One JSON line."""
    import torch
    from paper_1603_00937_b200 import build as gbe_build
    gbe_build.build()
    import paper_1603_00937_b200 as gbe
    s = make_system(args.workload, 0)
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = None if s.meta.get("kind") == "water" else torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    gbe.gbe_graph_set_sp2_path(g, 1)
    info = g.info
    D_full = torch.empty(info["nnz_D"], dtype=torch.float64, device="cuda")
    D_wave = torch.empty_like(D_full)
    ws = g.new_workspace()
    _, log = gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D_full)  # the sequence of this system
    seq = log.branch

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    reps = max(1, args.steps)
    t_full = timed(lambda: gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=ws, D_val=D_full,
                                                  want_log=False), reps)
    del ws
    torch.cuda.empty_cache()
    nbytes = max(int(args.waves_gb * 1e9) // 256 * 256, int(info["workspace_bytes_preset_min"]))
    wsb = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    t_wave = timed(lambda: gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=wsb, D_val=D_wave,
                                                  want_log=False), reps)
    cap = (nbytes - (info["workspace_bytes"] - 2 * ((info["dense_elems"] * 8 + 255) // 256 * 256))) // 2
    print(json.dumps({"waves": args.workload, "n": s.n, "n_part": s.n_part, "iters": int(len(seq)),
                      "workspace_full_gb": info["workspace_bytes"] * 1e-9, "workspace_bounded_gb": nbytes * 1e-9,
                      "workspace_min_gb": info["workspace_bytes_preset_min"] * 1e-9,
                      "waves_estimate": int(-(-info["dense_elems"] * 8 // max(1, cap))),
                      "ms_full": t_full, "ms_bounded": t_wave, "ratio": t_wave / t_full,
                      "bit_identical": bool(torch.equal(D_full, D_wave))}), flush=True)


def run_small(args) -> None:
    """Small systems (BASELINE.json configs[0] and relatives): the tiled kernels against the shared-memory-resident SP2
    kernel, one JSON line per (system, path): gbe_density eagerly, as a CUDA-graph replay, and gbe_density_preset
    without trace logging.  Times are CUDA-event means over 20 calls after 3 warm-ups, graph reused (as in MD)."""
    import torch
    from paper_1603_00937_b200 import build as gbe_build
    gbe_build.build()
    import gbe_inputs as gi
    import paper_1603_00937_b200 as gbe

    def mean_ms(fn, n=20):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    cases = [("config 1: chain, 512 orbitals, 16 communities", gi.config(1)),
             ("chain, 4736 orbitals, 148 communities", gi.chain(4736, 148, seed=1)),
             ("water box, 1536 orbitals, tau=1e-3, 128 communities", gi.water_box(256, 128, tau=1e-3)),
             ("banded, 14504 orbitals, 148 communities", gi.random_banded(14504, half_bw=6, n_part=148, seed=11, tau=1e-4, iters=40)),
             ("banded, 16872 orbitals, 148 communities", gi.random_banded(16872, half_bw=6, n_part=148, seed=11, tau=1e-4, iters=40)),
             ("banded, 1450 orbitals, 10 communities", gi.random_banded(1450, half_bw=6, n_part=10, seed=11, tau=1e-4, iters=40)),
             ("banded, 4608 orbitals, 32 communities", gi.random_banded(4608, half_bw=6, n_part=32, seed=11, tau=1e-4, iters=40)),
             ("banded, 9216 orbitals, 64 communities", gi.random_banded(9216, half_bw=6, n_part=64, seed=11, tau=1e-4, iters=40)),
             ("banded, 21312 orbitals, 148 communities", gi.random_banded(21312, half_bw=6, n_part=148, seed=11, tau=1e-4, iters=40)),
             ("chain, 19200 orbitals, 600 communities", gi.chain(19200, 600, seed=5)),
             ("banded, 58016 orbitals, 592 communities", gi.random_banded(58016, half_bw=6, n_part=592, seed=11, tau=1e-4, iters=40)),
             ("water box, 6144 orbitals, tau=1e-3, 256 communities", gi.water_box(1024, 256, tau=1e-3))]
    for name, s in cases:
        Hd = gbe.DeviceCSR.from_host(s.H)
        g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
        ws = g.new_workspace()
        D = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
        auto = {1: "tiled", 2: "resident", 3: "packed"}[int(g.info["sp2_path_chosen"])]
        seq = np.array([i & 1 for i in range(s.iters)], dtype=np.uint8)
        for path, pname in ((1, "tiled"), (2, "resident"), (3, "packed")):
            if path == 2 and not g.info["resident_fits"]:
                continue
            if path == 3 and not g.info["n_small"]:
                continue
            gbe.gbe_graph_set_sp2_path(g, path)
            if int(g.info["sp2_path_chosen"]) != path:  # e.g. resident requested, communities not co-resident
                continue
            n0 = gbe.gbe_launch_count()
            gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D, want_log=False)
            launches = gbe.gbe_launch_count() - n0
            eager = mean_ms(lambda: gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D, want_log=False))
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                torch.cuda.synchronize()
                cg = torch.cuda.CUDAGraph()
                with torch.cuda.graph(cg, stream=st):
                    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D, want_log=False, stream=st)
            replay = mean_ms(cg.replay)
            preset = mean_ms(lambda: gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=ws,
                                                            D_val=D, want_log=False))
            _, ph = gbe.gbe_density_timed(Hd, g, s.n_occ, s.iters, -1.0, workspace=ws, D_val=D)
            print(json.dumps({"small": name, "n": s.n, "n_part": s.n_part, "m_max": g.info["max_m"], "iters": s.iters,
                              "path": pname, "library_choice": auto, "cluster_exchange": int(g.info["resident_cluster"]) if path == 2 else 0, "launches_per_call": int(launches),
                              "density_eager_us": eager * 1e3, "density_graph_replay_us": replay * 1e3,
                              "preset_no_trace_eager_us": preset * 1e3,
                              "sp2_loop_us": (ph["x2_ms"] + ph["x2_last_ms"] + ph["trace_ms"]) * 1e3,
                              "orbitals_per_s_eager": s.n / (eager * 1e-3)}), flush=True)
        g.free()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="water4096", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="tau x partition sweep (BASELINE.json configs[4]) instead of the bench line")
    ap.add_argument("--sweep-out", default="", help="markdown table of the sweep")
    ap.add_argument("--fermi", action="store_true", help="time the finite-temperature Chebyshev expansion (Eq.(7)) instead")
    ap.add_argument("--fermi-order", type=int, default=60)
    ap.add_argument("--small", action="store_true", help="small systems: tiled kernels against the shared-memory-resident SP2 kernel")
    ap.add_argument("--gapped", action="store_true", help="sweep on the gapped variant of the water model, run to idempotency")
    ap.add_argument("--no-exact", action="store_true", help="sweep without the exact projector (no error columns)")
    ap.add_argument("--sweep-taus", default="", help="comma-separated thresholds of the sweep (default: the five of configs[4])")
    ap.add_argument("--sp2-path", type=int, default=0, help="sweep: force the SP2 kernels (1 tiled, 2 resident, 3 packed; 0 = the library's choice)")
    ap.add_argument("--waves", action="store_true", help="gbe_density_preset on the whole batch against the same call in a bounded workspace")
    ap.add_argument("--md", action="store_true", help="MD-like loop: Eq.(8) graph update + pre-set SP2 sequence + band energy per step")
    ap.add_argument("--md-tau", type=float, default=1e-4, help="--md: threshold on D(t - dt) in Eq.(8)")
    ap.add_argument("--timeline", default="", choices=["", "packed", "x2"],
                    help="in-kernel timeline of k_sp2_packed / k_x2_tma from %%globaltimer stamps (instrumented library copy)")
    ap.add_argument("--trace-build", action="store_true", help="timeline of one gbe_build_graph: device busy / idle time, gaps")
    ap.add_argument("--waves-gb", type=float, default=8.0, help="--waves: size of the bounded workspace in GB")
    ap.add_argument("--clock-sampler", default="nvml", choices=["nvml", "nvidia-smi", "none"],
                    help="how clocks / throttle reasons are sampled during the timed region (nvml: a thread of this process)")
    ap.add_argument("--record-traffic", default="", help="ncu raw-page CSV of a --set full capture of k_x2: write profiles/x2_traffic.json")
    ap.add_argument("--traffic-source", default="", help="the profiles/ summary that documents the capture")
    args = ap.parse_args()
    if args.record_traffic:
        record_traffic(args)
    elif args.sweep:
        run_sweep(args)
    elif args.small:
        run_small(args)
    elif args.waves:
        run_waves(args)
    elif args.trace_build:
        run_trace_build(args)
    elif args.timeline:
        run_timeline(args)
    elif args.md:
        run_md(args)
    elif args.fermi:
        run_fermi(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
