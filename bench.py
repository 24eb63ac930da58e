#!/usr/bin/env python
"""bench.py -- throughput of the f-x poststack depth-migration hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..3] [--impl ours|reference]
    python bench.py --sweep [--sweep-taps 15,25,51]     (configs[4], one JSON line per point)

A "step" is one pass of the whole hot path (table look-up, FIR extrapolation, depth marching,
imaging: SURVEY.md 8(a) A1-A7) over one f-x section: one `pdm_migrate` call.  At N = 1 the
workload is BASELINE.json configs[3] (the configuration the north_star target is quoted on);
inputs are seeded and synthetic.  Prints ONE JSON line on rank 0.

N > 1: weak scaling, one rank per GPU (launched by torchrun; `python bench.py --gpus N` without
torchrun re-executes itself under torch.distributed.run with N ranks, and fails loudly if the box
has fewer than N GPUs).  The job is the configs[3] model with an N-times denser frequency list (the
DFT bins of an N-times longer record); rank r owns the bins offset by r/N (803 lines each,
frequencies are independent units) and the partial images are summed with one NCCL
all-reduce inside the timed step -- the path's only exchange.

--impl reference: times the FP64 CPU oracle (oracle/, as it stands) on the host cores on a
bounded sample of the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "extrapolated samples/sec (z*omega*x points/s)"
UNIT = "samples/s"
# FP32 peak the guide's unit counts and clocks give: 148 SMs x 128 FP32
# lanes x 2 flop/FMA x 1.965 GHz max SM clock.  The FFMA-chain microbenchmark (pdm_fp32_peak)
# reads 71-73 TFLOP/s on this pool; both are reported.
FP32_PEAK_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r03_traffic.json")


def csrc_digest() -> str:
    """sha1 over the kernel sources: ties an ncu traffic figure to the code it was captured on."""
    import hashlib
    d = os.path.join(ROOT, "paper_1912_05529_b200", "csrc")
    h = hashlib.sha1()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            with open(os.path.join(d, name), "rb") as f:
                h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(config: int, path: str, flags: int, world: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
    committed `ncu --set full` capture (profiles/r03_traffic.json) -- only when that capture was
    taken on exactly these kernel sources, this config and this path; else None with the reason."""
    if world != 1 or flags:
        return None, "no capture for multi-rank runs / non-default flags"
    try:
        with open(TRAFFIC_FILE) as f:
            table = json.load(f)
    except (OSError, ValueError):
        return None, "profiles/r03_traffic.json absent"
    for e in table.get("captures", []):
        if e.get("config") == config and e.get("path") == path:
            if e.get("csrc_sha1") != csrc_digest():
                return None, (f"capture {e.get('report')} was taken on csrc {e.get('csrc_sha1')}, "
                              f"HEAD is {csrc_digest()}: stale")
            return float(e["dram_bytes_read"]) + float(e["dram_bytes_write"]), e.get("report")
    return None, "no capture for this config/path"


def load_workload(k: int, rank: int, world: int) -> dict:
    import pdm_inputs
    if k == 3:
        from pdm_inputs.configs import config3_rank_shard
        return config3_rank_shard(rank, world)
    cfg = pdm_inputs.make_config(k)
    if world > 1:                        # small configs: plain round-robin shard of the lines
        from paper_1912_05529_b200.shard import shard_workload
        cfg = shard_workload(cfg, rank, world)
    return cfg


def workload_name(k: int, cfg: dict, world: int) -> str:
    s = (f"configs[{k}] nx={cfg['nx']} nz={cfg['nz']} nw={cfg['nw']} taps={cfg['ntaps']} "
         f"ntab={cfg['ntab']}")
    if world > 1:
        s += f" per rank x {world} ranks (frequency-sharded, image all-reduce)"
    return s


def bench_config(k: int, cfg: dict, world: int) -> dict:
    """The `config` object, identical in both arms (launch details of our arm go under `launch`)."""
    return {"workload": workload_name(k, cfg, world),
            "l2": "GPU arm: 256 MiB buffer written between timed steps (L2 flush), CUDA events on the launching "
                  "stream; reference arm: the FP64 oracle on the host cores, wall clock"}


def executed_frac(info: dict, seconds: float) -> float:
    """FP32 lane-operations the kernels actually execute (pdm_info.executed_lane_ops: folded taps counted
    once, zero-padded taps counted) x 2 flop / time / the derived FP32 peak -- beside the COUNTED fraction,
    whose ratio to this one differs per kernel family (1.32 folded 1-D, 1.0 general, 2.45 folded 15x15 3-D)."""
    return info["executed_lane_ops"] * 2.0 / seconds / (FP32_PEAK_NOMINAL_TFLOPS * 1e12)


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)),
                "sm_min_mhz": float(min(sm)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------- oracle legs
def oracle_sample(cfg: dict, lines_per_thread: int = 4):
    """Time the FP64 oracle, as it stands, on a bounded sample: `lines_per_thread` x threads
    evenly spaced frequency lines of the workload, all nz depth steps, all nx samples."""
    import oracle
    oracle.build()
    threads = oracle.num_threads()
    n = min(cfg["nw"], max(1, lines_per_thread * threads))
    idx = np.unique(np.linspace(0, cfg["nw"] - 1, n).round().astype(np.int32))
    t0 = time.perf_counter()
    oracle.migrate(cfg, omega_index=idx)
    dt = time.perf_counter() - t0
    samples = float(idx.size) * cfg["nx"] * cfg["nz"]
    return samples / dt, dt, int(idx.size), threads


def run_reference(args, rank: int, world: int):
    if rank != 0:
        return
    cfg = load_workload(args.config, 0, 1)
    import oracle
    # per-step sample: 4 lines per thread (the cpu_baseline leg of our arm takes 16, once): large enough that
    # the oracle's fixed costs (q map, per-thread image accumulators) no longer depress the rate, small
    # enough that warmup + steps stay within a few minutes at configs[3] (~3 s per step on 16 cores)
    threads = oracle.num_threads()
    times, sps = [], []
    for i in range(args.warmup + args.steps):
        v, dt, nlines, threads = oracle_sample(cfg, lines_per_thread=args.ref_lines_per_thread)
        if i >= args.warmup:
            times.append(dt); sps.append(v)
    value = float(np.mean(sps))
    sample = (f"{nlines} evenly spaced omega lines of {cfg['nw']} per step, all nz={cfg['nz']} depth "
              f"steps, all nx={cfg['nx']} samples")
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic", "config": bench_config(args.config, cfg, 1),
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                            "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------- our arm
PATH_NAMES = {1: "smem-marching", 2: "x-tiled", 3: "naive", 4: "cluster", 5: "packed"}


def time_migrate(plan, P0, image, stream, flush, torch, steps: int, warmup: int = 3):
    """ms of `steps` pdm_migrate calls (CUDA events on the launching stream, L2 flushed between)."""
    for _ in range(warmup):
        plan.migrate(P0, image, stream=stream)
    torch.cuda.synchronize()
    ms = []
    for _ in range(steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        plan.migrate(P0, image, stream=stream)
        b.record(stream)
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    return ms


def oracle_one_thread(k: int, max_lines: int = 12):
    """the oracle on ONE host thread for the small configs (a fresh process with
    OMP_NUM_THREADS=1; a bounded sample of evenly spaced lines) -> samples/s, or None."""
    code = (f"import sys, time, json, numpy as np; sys.path.insert(0, {ROOT!r}); import oracle, pdm_inputs;"
            f"c = pdm_inputs.make_config({k}); n = min(c['nw'], {max_lines});"
            "idx = np.unique(np.linspace(0, c['nw'] - 1, n).round().astype(np.int32));"
            "oracle.migrate(c, omega_index=idx[:1]); t = time.perf_counter(); oracle.migrate(c, omega_index=idx);"
            "dt = time.perf_counter() - t;"
            "print(json.dumps({'v': float(idx.size) * c['nx'] * c['nz'] / dt, 'lines': int(idx.size), 'threads': oracle.num_threads()}))")
    try:
        out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, OMP_NUM_THREADS="1"),
                             capture_output=True, text=True, timeout=300)
        return json.loads(out.stdout.strip().splitlines()[-1])
    except Exception:                                       # a reported baseline only: never fail the bench over it
        return None


def other_configs(pdm, torch, dev, stream, flush):
    """The regimes the headline workload does not show, measured in the same run (a few seconds):
    configs[0..2] and two configs[4] points where every sample has its own table row (tap-gather
    bound) -- ms per migrate and the counted FP32 fraction, so that these are driver-measured too."""
    import pdm_inputs
    from pdm_inputs.configs import sweep_point
    work = [(f"configs[{k}]", (lambda k=k: pdm_inputs.make_config(k))) for k in (0, 1, 2)]
    work += [("configs[4] field", lambda: sweep_point(32768, 1024, 15)),
             ("configs[4] field", lambda: sweep_point(4096, 1024, 51))]
    rows = []
    for name, make in work:
        cfg = make()
        with pdm.Plan.from_config(cfg, 0) as plan:
            info = plan.info
            P0 = torch.from_numpy(cfg["P0"]).to(dev)
            image = torch.empty((cfg["nz"], cfg["nx"]), dtype=torch.float32, device=dev)
            ms = time_migrate(plan, P0, image, stream, flush, torch, steps=5)
        t = float(np.median(ms)) * 1e-3
        sps = info["samples"] / t
        rows.append({"workload": f"{name} nx={cfg['nx']} nz={cfg['nz']} nw={cfg['nw']} taps={cfg['ntaps']}",
                     "path": PATH_NAMES[info["path"]], "ms_median": t * 1e3, "ms_best": float(min(ms)),
                     "samples_per_s": sps,
                     "frac_fp32_peak_counted": sps * 8 * cfg["ntaps"] / (FP32_PEAK_NOMINAL_TFLOPS * 1e12),
                     "frac_fp32_peak_executed": executed_frac(info, t),
                     "frac_hbm_16B_per_sample_of_measured":
                         (sps * 16 / (measured_hbm_gbs()[0] * 1e9)) if info["path"] == pdm.PDM_PATH_TILED else None})
        if name in ("configs[0]", "configs[1]"):
            o = oracle_one_thread(int(name[8]))
            if o:
                rows[-1]["oracle_one_thread"] = {"value": o["v"], "unit": UNIT, "cores": o["threads"],
                                                 "sample": f"{o['lines']} evenly spaced omega lines"}
        del P0, image
    return rows


def run_ours(args, rank: int, local_rank: int, world: int):
    import torch
    import torch.distributed as dist

    import paper_1912_05529_b200 as pdm
    from paper_1912_05529_b200.shard import allreduce_image

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    pdm.load_library()                      # raises if libpdm.so was not built
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    print(f"[bench] rank {rank} of {world} on cuda:{local_rank} ({torch.cuda.get_device_name(local_rank)})",
          file=sys.stderr, flush=True)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")        # communicator log: shows the N ranks (and NVLS)
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=dev)

    cfg = load_workload(args.config, rank, world)
    t_create = time.perf_counter()
    plan = pdm.Plan.from_config(cfg, args.flags)          # pdm_create: excluded from the metric, reported
    torch.cuda.synchronize(dev)
    create_ms = 1e3 * (time.perf_counter() - t_create)
    info = plan.info
    samples = info["samples"]
    stream = torch.cuda.current_stream(dev)

    P0 = torch.from_numpy(cfg["P0"]).to(dev)
    image = torch.empty((cfg["nz"], cfg["nx"]), dtype=torch.float32, device=dev)
    P0_pinned = torch.from_numpy(cfg["P0"]).pin_memory()
    image_pinned = torch.empty((cfg["nz"], cfg["nx"]), dtype=torch.float32).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step():
        plan.migrate(P0, image, stream=stream)
        if world > 1:
            allreduce_image(image)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    plan.profile(True)
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    # ---- device-resident timing: K steps, CUDA events on the launching stream, L2 flushed between
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    main_ms, reduce_ms = [], []
    barrier()
    for a, b in ev:
        flush.zero_()                                    # L2 flush, outside the timed pair
        a.record(stream)
        step()
        b.record(stream)
        m, r = plan.profile_read()                       # syncs on this step's last kernel event
        main_ms.append(m); reduce_ms.append(r)
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = torch.tensor([float(sum(step_ms))], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    plan.profile(False)

    # ---- end to end through the public HOST-buffer call (pinned host memory, copies inside)
    h2d = cfg["P0"].nbytes
    d2h = image_pinned.numel() * 4
    plan.migrate_host(P0_pinned, image_pinned, stream=stream)
    barrier()
    e2e_ev = []
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        plan.migrate_host(P0_pinned, image_pinned, stream=stream)   # returns after the D2H copy
        if world > 1:
            # the reduced image is what the job returns: reduce on device, then read it back
            image.copy_(image_pinned, non_blocking=True)
            allreduce_image(image)
            image_pinned.copy_(image, non_blocking=True)
        b.record(stream)
        e2e_ev.append((a, b))
    barrier()
    e2e_ms = torch.tensor([float(sum(a.elapsed_time(b) for a, b in e2e_ev))],
                          dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_ms, op=dist.ReduceOp.MAX)
    e2e_ms = float(e2e_ms.item())
    clocks = sampler.stop()

    if rank == 0:
        k = args.steps
        value = samples * world * k / (total_ms * 1e-3)
        main_avg = float(np.mean(main_ms))
        launches_main = info["launches_per_migrate"] - 1 if info["path"] != pdm.PDM_PATH_NAIVE else info["launches_per_migrate"]
        per_launch_ms = main_avg / max(1, launches_main)
        flops_per_launch = info["counted_flops"] / max(1, launches_main)
        achieved = flops_per_launch / (per_launch_ms * 1e-3) / 1e12
        try:
            fma_peak = pdm.pdm_fp32_peak(True, 50000, 3, stream.cuda_stream)
        except pdm.PdmError:
            fma_peak = None
        kernel = {pdm.PDM_PATH_SMEM: "pdm_march_kernel", pdm.PDM_PATH_TILED: "pdm_tiled_step",
                  pdm.PDM_PATH_NAIVE: "pdm_naive_step", pdm.PDM_PATH_CLUSTER: "pdm_cluster_kernel",
                  pdm.PDM_PATH_PACKED: "pdm_pack_kernel"}[info["path"]]
        path_name = PATH_NAMES[info["path"]]
        traffic, traffic_src = ncu_traffic(args.config, path_name, args.flags, world)
        algo_bytes = float(cfg["P0"].nbytes + 4 * cfg["nz"] * cfg["nx"] + cfg["velocity"].nbytes)
        roofline = {"bound": "alu", "kernel": kernel, "achieved": achieved,
                    "peak": FP32_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                    "frac": achieved / FP32_PEAK_NOMINAL_TFLOPS,
                    "frac_executed": executed_frac(info, main_avg * 1e-3),
                    "traffic": traffic,
                    "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                    "traffic_source": traffic_src,
                    "algorithmic_bytes": algo_bytes,
                    "algorithmic_bytes_are": "P0 in + q map once + image out (the wavefield never leaves the SM)",
                    "traffic_over_algorithmic": (traffic / algo_bytes) if traffic else None,
                    "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md); "
                                   "MEASURED_PEAKS.json has no FP32 entry",
                    "ffma_chain_measured_tflops": fma_peak,
                    "frac_of_ffma_chain": (achieved / fma_peak) if fma_peak else None,
                    "flops_counted": "8*(2L+1) per sample (metric definition); the kernel folds "
                                     "W_k == W_-k and executes (6L+4)/(4(2L+1)) of the lane-ops",
                    "kernel_ms_per_launch": per_launch_ms, "launches_per_step": launches_main,
                    "kernel_share_of_step": main_avg / (float(np.mean(step_ms))),
                    "reduce_ms": float(np.mean(reduce_ms))}
        cpu_v, cpu_dt, cpu_lines, cpu_threads = oracle_sample(cfg, lines_per_thread=args.cpu_lines_per_thread)
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": k,
               "warmup": max(args.warmup, 3), "ms_per_step": total_ms / k,
               "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_best": float(min(step_ms)),
               "create_ms": create_ms, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
               "config": bench_config(args.config, cfg, world),
               "launch": {"path": path_name, "grid": f"{info['grid_ctas']}x{info['threads_per_cta']}",
                          "smem_bytes": info["smem_bytes"], "workspace_gb": info["workspace_bytes"] / 1e9},
               "pct_fp32_peak_counted": 100.0 * value / world * 8 * cfg["ntaps"] / (FP32_PEAK_NOMINAL_TFLOPS * 1e12),
               "roofline": roofline,
               "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cpu_threads, "kind": "oracle",
                                "sample": f"{cpu_lines} evenly spaced omega lines of {cfg['nw']}, all "
                                          f"nz={cfg['nz']} steps, all nx={cfg['nx']} samples, "
                                          f"{cpu_dt:.1f} s wall"},
               "e2e": {"value": samples * world * k / (e2e_ms * 1e-3), "unit": UNIT,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                       "ms_per_step": e2e_ms / k},
               "gpu_launches": int(info["launches_per_migrate"]) * k,
               "clocks": clocks}
        if world == 1 and not args.no_extra:
            import copy
            a2 = copy.copy(args)
            a2.flags, a2.steps = 0, min(args.steps, 5)
            out["extra"] = {"other_configs": other_configs(pdm, torch, dev, stream, flush),
                            # the stages around / beyond the poststack hot path, same run
                            "other_stages": measure_tf(a2) + measure_design(a2) + measure_prestack(a2) + measure_3d(a2)}
        print(json.dumps(out), flush=True)
    plan.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------------------- configs[4] sweep
SWEEP_NX = (1024, 4096, 16384, 32768)
SWEEP_NW = (64, 256, 1024, 2048)
SWEEP_TAPS = (15, 25, 51)


def measured_hbm_gbs():
    """(GB/s, source): the driver-measured copy bandwidth, else the profiling guide's fallback."""
    for cand in ("/root/repo/MEASURED_PEAKS.json", os.path.join(ROOT, "MEASURED_PEAKS.json")):
        if os.path.exists(cand):
            with open(cand) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def run_sweep(args):
    """BASELINE.json configs[4]: samples/s and roofline fraction per (nx, nw, taps) point, one JSON
    line each (parity of sampled points is tests/test_gpu_parity.py's job, not this loop's)."""
    import torch

    import paper_1912_05529_b200 as pdm
    from pdm_inputs.configs import sweep_point

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    pdm.load_library()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    hbm_gbs, hbm_src = measured_hbm_gbs()
    def pick(arg, full):
        return tuple(int(t) for t in arg.split(",")) if arg else full
    for ntaps in pick(args.sweep_taps, SWEEP_TAPS):
        for nx in pick(args.sweep_nx, SWEEP_NX):
            for nw in pick(args.sweep_nw, SWEEP_NW):
                cfg = sweep_point(nx, nw, ntaps, model=args.sweep_model)
                try:
                    plan = pdm.Plan.from_config(cfg, args.flags)
                except pdm.PdmError as e:             # a forced kernel form that cannot run this point
                    print(json.dumps({"workload": f"configs[4] nx={nx} nz={cfg['nz']} nw={nw} taps={ntaps} "
                                                  f"velocity={args.sweep_model}", "error": str(e)}), flush=True)
                    continue
                info = plan.info
                P0 = torch.from_numpy(cfg["P0"]).to(dev)
                image = torch.empty((cfg["nz"], nx), dtype=torch.float32, device=dev)
                steps = int(max(2, min(args.steps, 4e10 // info["samples"])))
                for _ in range(3):
                    plan.migrate(P0, image, stream=stream)
                torch.cuda.synchronize(dev)
                ms = []
                for _ in range(steps):
                    flush.zero_()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    plan.migrate(P0, image, stream=stream)
                    b.record(stream)
                    torch.cuda.synchronize(dev)
                    ms.append(a.elapsed_time(b))
                t = float(np.median(ms)) * 1e-3
                sps = info["samples"] / t
                tiled = info["path"] == pdm.PDM_PATH_TILED
                out = {"workload": f"configs[4] nx={nx} nz={cfg['nz']} nw={nw} taps={ntaps} velocity={args.sweep_model}",
                       "path": PATH_NAMES[info["path"]],
                       "taps_mode": info["taps_mode"], "grid": f"{info['grid_ctas']}x{info['threads_per_cta']}",
                       "launches": info["launches_per_migrate"], "steps": steps, "ms": t * 1e3,
                       "samples_per_s": sps,
                       "frac_fp32_peak_counted": sps * 8 * ntaps / (FP32_PEAK_NOMINAL_TFLOPS * 1e12),
                       "frac_fp32_peak_executed": executed_frac(info, t),
                       "frac_hbm_16B_per_sample": (sps * 16 / (hbm_gbs * 1e9)) if tiled else None,
                       "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": hbm_src}
                print(json.dumps(out), flush=True)
                plan.close()
                del P0, image


# ------------------------------------------------------------------------------- t -> f transform
def measure_tf(args):
    """the time -> frequency transform of the input section at configs[3]'s size
    (nt = 4096 samples, nx = 6144 traces, the 803 bins of 2-100 Hz), one JSON line."""
    import torch

    import paper_1912_05529_b200 as pdm
    from pdm_inputs.configs import dft_bin_omegas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    pdm.load_library()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream(dev)
    nt, dt, nx = 4096, 0.002, 6144
    omega = dft_bin_omegas(nt, dt, 2.0, 100.0)
    bins = np.rint(np.asarray(omega, np.float64) * nt * dt / (2 * np.pi)).astype(np.int32)
    section = torch.randn((nt, nx), dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    with pdm.SectionTransform(nt, nx, bins) as tf:
        out = tf.forward(section)
        for _ in range(max(args.warmup, 3)):
            tf.forward(section, out=out, stream=stream)
        torch.cuda.synchronize(dev)
        ms = []
        for _ in range(args.steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            tf.forward(section, out=out, stream=stream)
            b.record(stream)
            torch.cuda.synchronize(dev)
            ms.append(a.elapsed_time(b))
    t = float(np.median(ms)) * 1e-3
    # nt is a power of two here: the library runs a real FFT per trace (kern_fft.cuh), bound by moving
    # the section in and the band's bins out once; the contraction form (other nt) is FP32-bound
    hbm_gbs, hbm_src = measured_hbm_gbs()
    algo_bytes = 4.0 * nt * nx + 8.0 * bins.size * nx
    return [({"workload": f"t->f transform nt={nt} nx={nx} nw={bins.size} (configs[3] record)",
                      "kernel": "pdm_fft_kernel", "steps": args.steps, "ms": t * 1e3, "ms_best": float(min(ms)),
                      "bin_trace_outputs_per_s": bins.size * nx / t,
                      "roofline": {"bound": "hbm", "achieved": algo_bytes / t / 1e9, "peak": hbm_gbs,
                                   "unit": "GB/s", "frac": algo_bytes / t / 1e9 / hbm_gbs,
                                   "peak_source": hbm_src, "algorithmic_bytes": algo_bytes,
                                   "algorithmic_bytes_are": "section in (4 B x nt x nx) + P0 out (8 B x nw x nx)"},
                      "contraction_equivalent_tflops": 4.0 * nt * bins.size * nx / t / 1e12,
                      "share_of_migration": "compare ms with bench.py's ms_per_step on configs[3]"})]


# ------------------------------------------------------------------------------- table design
def measure_design(args):
    """pdm_design_table for configs[3]'s table (1024 rows x 51 taps, 200 D2 sweeps on a
    2048-point grid, FP64) -- a synchronous setup call, so wall clock around it (median of 3 after one warm-up)."""
    import torch

    import paper_1912_05529_b200 as pdm

    pdm.load_library()
    torch.cuda.set_device(0)
    ntab, ntaps, du = 1024, 51, 4.19 / 1023
    pdm.pdm_design_table(16, ntaps, du, 1.0)
    torch.cuda.synchronize()
    ts = []
    for _ in range(3):
        t0 = time.perf_counter()
        pdm.pdm_design_table(ntab, ntaps, du, 1.0)
        ts.append(time.perf_counter() - t0)
    t = float(np.median(ts))
    # per row and sweep: forward (N/2+1) x (L+1) + inverse (L+1) x (N/2+1) FP64 multiply-adds on the half grid
    fma = 2.0 * 200 * ntab * (1024 + 1) * 26
    return [{"workload": f"table design ntab={ntab} taps={ntaps} (configs[3]'s table), 200 sweeps, grid 2048, FP64",
             "kernel": "pdm_design_kernel", "steps": 3, "ms": t * 1e3, "ms_best": float(min(ts)) * 1e3,
             "rows_per_s": ntab / t, "fp64_tflops": 2.0 * fma / t / 1e12,
             "includes": "host validation, cosine-table upload, kernel, D2H copy of the table (synchronous call)"}]


# ------------------------------------------------------------------------------- prestack shot
def measure_prestack(args):
    """one prestack shot (pdm_migrate_shot) on a configs[4] field point -- both
    wavefields are extrapolated, so a shot counts 2 x nx x nz x nw extrapolated samples."""
    import torch

    import paper_1912_05529_b200 as pdm
    from pdm_inputs.configs import sweep_point

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    pdm.load_library()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    nx, nw, ntaps = 4096, 1024, 25
    cfg = sweep_point(nx, nw, ntaps)
    rec = torch.from_numpy(cfg["P0"]).to(dev)
    src = torch.roll(rec, 1, 0).contiguous()
    image = torch.empty((cfg["nz"], nx), dtype=torch.float32, device=dev)
    with pdm.Plan.from_config(cfg, pdm.PDM_PRESTACK | args.flags) as plan:
        info = plan.info
        for _ in range(max(args.warmup, 3)):
            plan.migrate_shot(src, rec, image, stream=stream)
        torch.cuda.synchronize(dev)
        ms = []
        for _ in range(args.steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            plan.migrate_shot(src, rec, image, stream=stream)
            b.record(stream)
            torch.cuda.synchronize(dev)
            ms.append(a.elapsed_time(b))
    t = float(np.median(ms)) * 1e-3
    sps = info["samples"] / t
    return [({"workload": f"prestack shot, configs[4] field nx={nx} nz={cfg['nz']} nw={nw} taps={ntaps} "
                                  "(2 wavefields per frequency)", "kernel": "pdm_pack_kernel (xcorr)",
                      "path": PATH_NAMES[info["path"]], "grid": f"{info['grid_ctas']}x{info['threads_per_cta']}",
                      "steps": args.steps, "ms": t * 1e3, "ms_best": float(min(ms)), "samples_per_s": sps,
                      "frac_fp32_peak_counted": sps * 8 * ntaps / (FP32_PEAK_NOMINAL_TFLOPS * 1e12),
                      "frac_fp32_peak_executed": executed_frac(info, t)})]


# ------------------------------------------------------------------------------- 3-D variant
def measure_3d(args):
    """the 3-D variant (2-D extrapolators) on seeded 256 x 256 x 64 volumes,
    64 frequencies; one JSON line per (operator size, velocity model).  Counted flops: 8 x ntaps^2 per sample."""
    import torch

    import paper_1912_05529_b200 as pdm
    import pdm_inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    pdm.load_library()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    nx = ny = 256; nz = 64; nw = 64
    rows = []
    for ntaps, model, sym in ((7, "layers", False), (7, "field", False), (15, "layers", False), (15, "field", False),
                              (7, "layers", True), (15, "layers", True), (15, "field", True), (15, "field", "designed")):
        if True:
            cfg = pdm_inputs.random_problem_3d(5, nx, ny, nz, nw, ntaps, model=model, symmetric=bool(sym))
            if sym == "designed":           # 2-D extrapolators from the designed 1-D rows (McClellan transformation)
                from pdm_inputs import filters
                cfg["table"] = filters.mcclellan_table(filters.design_table(cfg["ntab"], ntaps, cfg["du"], 1.0))
            P0 = torch.from_numpy(cfg["P0"]).to(dev)
            image = torch.empty((nz, ny, nx), dtype=torch.float32, device=dev)
            with pdm.Plan3D.from_config(cfg, args.flags) as plan:
                info = plan.info
                for _ in range(max(args.warmup, 3)):
                    plan.migrate(P0, image, stream=stream)
                torch.cuda.synchronize(dev)
                ms = []
                for _ in range(args.steps):
                    flush.zero_()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    plan.migrate(P0, image, stream=stream)
                    b.record(stream)
                    torch.cuda.synchronize(dev)
                    ms.append(a.elapsed_time(b))
            t = float(np.median(ms)) * 1e-3
            sps = info["samples"] / t
            hbm_gbs, _ = measured_hbm_gbs()
            rows.append(({"workload": f"3-D nx={nx} ny={ny} nz={nz} nw={nw} taps={ntaps}x{ntaps} velocity={model}"
                                      + (" operator symmetric in kx, ky (folded kernels)" if sym else "")
                                      + (", McClellan-designed table" if sym == "designed" else ""),
                              "kernel": "pdm3_step", "grid": f"{info['grid_ctas']}x{info['threads_per_cta']}",
                              "smem_bytes": info["smem_bytes"], "steps": args.steps, "ms": t * 1e3,
                              "ms_best": float(min(ms)), "samples_per_s": sps,
                              "frac_fp32_peak_counted": sps * 8 * ntaps * ntaps / (FP32_PEAK_NOMINAL_TFLOPS * 1e12),
                              "frac_fp32_peak_executed": executed_frac(info, t),
                              "frac_hbm_16B_per_sample": sps * 16 / (hbm_gbs * 1e9)}))
    return rows


def run_tf(args):
    for row in measure_tf(args):
        print(json.dumps(row), flush=True)


def run_prestack(args):
    for row in measure_prestack(args):
        print(json.dumps(row), flush=True)


def run_3d(args):
    for row in measure_3d(args):
        print(json.dumps(row), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3])
    ap.add_argument("--flags", type=lambda s: int(s, 0), default=0, help="pdm_create flags word")
    ap.add_argument("--cpu-lines-per-thread", type=int, default=16)
    ap.add_argument("--ref-lines-per-thread", type=int, default=4,
                    help="--impl reference: omega lines per host thread and step")
    ap.add_argument("--no-extra", action="store_true",
                    help="skip extra.other_configs (configs[0..2] + two configs[4] points, N = 1 only)")
    ap.add_argument("--tf", action="store_true", help="time the t->f transform of the section (SURVEY 8(f) N1)")
    ap.add_argument("--3d", dest="three_d", action="store_true", help="time the 3-D variant (SURVEY 8(f) N4)")
    ap.add_argument("--prestack", action="store_true", help="time one prestack shot (SURVEY 8(f) N4)")
    ap.add_argument("--sweep", action="store_true", help="configs[4] throughput sweep, one JSON line per point")
    ap.add_argument("--sweep-taps", default="", help="comma list of tap counts to sweep (default 15,25,51)")
    ap.add_argument("--sweep-nx", default="", help="comma list of nx (default 1024,4096,16384,32768)")
    ap.add_argument("--sweep-nw", default="", help="comma list of nw (default 64,256,1024,2048)")
    ap.add_argument("--sweep-model", default="field", choices=["field", "layers"],
                    help="velocity of the sweep: BASELINE.json's random field, or flat layers "
                         "(warp-uniform table rows: the HBM-bound regime of the x-tiled path)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    multi = not (args.tf or args.sweep or args.prestack or args.three_d)
    if multi and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the N ranks ourselves (one process per GPU, NCCL), loudly
        # refusing a box with fewer GPUs -- never a silent 1-rank run that prints n_gpus: 1
        if args.impl == "ours":
            import torch
            have = torch.cuda.device_count()
            if have < args.gpus:
                raise SystemExit(f"bench.py: --gpus {args.gpus} but this box has {have} CUDA device(s)")
        import socket
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                  f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
                                  "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]])
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if multi and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU")
    if args.tf:
        if rank == 0:
            run_tf(args)
    elif args.three_d:
        if rank == 0:
            run_3d(args)
    elif args.prestack:
        if rank == 0:
            run_prestack(args)
    elif args.sweep:
        if rank == 0:
            run_sweep(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
