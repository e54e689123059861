#!/usr/bin/env python
"""bench.py -- throughput of the VRC ray-cast hot path on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

A "step" is one pass of the whole hot path over one batch of synthetic rays: S1 cross sections ->
S2/S3 mesh walk -> S4/S5 Eq. (4) score -> S6 fp64 tally accumulation (mr_cast_rays).  The default
workload is BASELINE.json configs[2], the PWR 17x17-like lattice (170x170x300 cells, K = 3,
10^7 rays per batch): the configuration north_star's roofline target is quoted on.

  value   : whole-job ray-cell segments/s with the ray batch already resident in HBM
  e2e     : the same metric through the C ABI with HOST buffers: each step copies the batch from
            pinned host memory (mr_cast_rays, where = host) and reads the tally back (mr_read_tally)
  roofline: ALGORITHMIC bytes (31 B/segment + 96 B/ray on this config) / cast-kernel time, against
            the measured copy bandwidth in MEASURED_PEAKS.json.  `achieved` is that algorithmic rate, NOT DRAM traffic
            (the working set is L2-resident): the DRAM rate from the committed ncu capture, the unit that really
            limits the kernel, the measured L2 fp64-atomic ceiling and the whole-step fraction (ordering pre-pass
            included) are reported beside it, and `roofline_plain_records` repeats the figure with the dictionary /
            tiled-index path switched off (what a mesh with many distinct cell records gets)
  cpu_baseline: the CPU oracle, as it stands, on the box's host cores over a bounded sample

    python bench.py --microbench red     the L2 fp64-atomic micro-benchmark alone (mr_microbench_red)

N > 1 (torchrun, one rank per GPU): every rank holds the whole problem and casts its own batches
(weak scaling, no data-path collective); time = max over ranks.  --impl reference times the
oracle on the host cores (rank 0 only).
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

METRIC = "ray_cell_segments_per_sec"
UNIT = "segments/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def algorithmic_bytes(prob, segments: int, rays: int, dense: bool = False) -> int:
    """B_seg = 16 + 5K (dense: 16 + 4K), B_ray = 32 + 16 M (mixed mode)."""
    b_seg = 16 + (4 if dense else 5) * prob.K
    b_ray = 32 + 16 * prob.M
    return segments * b_seg + rays * b_ray


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


TRAFFIC_SOURCES = {}


def committed_profile(workload: str, kernel: str):
    """(dram bytes per launch, limiter dict) of `kernel` on `workload` from the committed ncu captures
    (profiles/traffic.txt: `workload kernel dram_bytes commit`; profiles/limiters.json), or (None, None)."""
    traffic, limiter = None, None
    try:
        for line in open(os.path.join(ROOT, "profiles", "traffic.txt")):
            w = line.split()
            if len(w) >= 3 and not line.startswith("#") and w[0] == workload and w[1] == kernel:
                traffic = float(w[2])
                TRAFFIC_SOURCES[f"{workload}:{kernel}"] = " ".join(w[3:])   # commit and capture the figure comes from
    except OSError:
        pass
    try:
        with open(os.path.join(ROOT, "profiles", "limiters.json")) as f:
            limiter = json.load(f).get(f"{workload}:{kernel}")
    except (OSError, ValueError):
        pass
    return traffic, limiter


def run_microbench(args):
    """--microbench red: random fp64 red.global.add into an array the size of the PWR tally (69 MB, L2-resident), alone
    and paired with a 16- / 32-byte gather from the same cell, lanes in groups of 1/2/4/8 sharing consecutive cells."""
    import torch

    from paper_1706_07476_b200 import microbench_red

    if not torch.cuda.is_available():
        raise SystemExit("the micro-benchmark needs a CUDA device")
    rows = []
    for ncell in (8_670_000, 1_000_000, 134_217_728):
        for gather in (0, 16, 32):
            for group in (1, 2, 4, 8):
                r = microbench_red(0, ncell, group, gather, 1 << 28, 5)
                rows.append(r)
                print(f"# ncell {ncell:>10} gather {gather:>2} B group {group}: {r['best_ms']:.3f} ms "
                      f"{r['lane_ops_per_sec'] / 1e9:7.1f} G lane-ops/s", file=sys.stderr)
    print(json.dumps({"microbench": "red", "unit": "lane-ops/s", "rows": rows}))
    return 0


class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while `active` (the timed regions)."""

    def __init__(self, cuda_index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.active = False
        self._stop = False
        self._thread = None
        try:
            import pynvml
            import torch

            pynvml.nvmlInit()
            try:
                uuid = str(torch.cuda.get_device_properties(cuda_index).uuid)
                uuid = uuid if uuid.startswith("GPU-") else "GPU-" + uuid
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(cuda_index)
            self.nv = pynvml
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        except Exception as e:  # no NVML: report that instead of numbers
            self.error = repr(e)

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop:
            if self.active:
                try:
                    self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                    try:
                        mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                    except Exception:
                        mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                    for bit, nm in names.items():
                        if mask & bit:
                            self.reasons.add(nm)
                except Exception:
                    pass
            time.sleep(0.01)

    def report(self):
        self._stop = True
        if self._thread is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": getattr(self, "error", "nvml unavailable")}
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def cpu_oracle_rate(prob, rays, threads: int):
    """segments/s of the oracle as it stands on `threads` host threads over `rays`."""
    from oracle.vrc_oracle import Oracle

    orc = Oracle(prob)
    t0 = time.perf_counter()
    res = orc.cast(rays, threads=threads)
    dt = time.perf_counter() - t0
    return res.segments / dt, res.segments, dt, res.threads


def run_reference(args, prob_kw):
    """--impl reference: the CPU oracle on a bounded sample of the same workload, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle.vrc_oracle import Oracle, max_threads
    from workloads import CONFIG_NAMES, make_problem, make_rays

    prob = make_problem(args.config, **prob_kw)
    threads = max(1, min(max_threads(), len(os.sched_getaffinity(0))))
    n_sample = args.ref_rays
    rays = make_rays(prob, n_sample)
    orc = Oracle(prob)
    for _ in range(args.warmup):
        orc.cast(rays[: max(1000, n_sample // 10)], threads=threads)
    t0 = time.perf_counter()
    segs = 0
    for _ in range(args.steps):
        segs += orc.cast(rays, threads=threads).segments
    dt = time.perf_counter() - t0
    value = segs / dt
    sample = f"{n_sample} rays ({segs // args.steps} segments) of the workload per step, all host threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": CONFIG_NAMES[args.config], "reference": "CPU oracle (oracle/vrc_oracle.c), host cores",
                   "rays_per_step": n_sample},
        "rays_per_sec": n_sample * args.steps / dt,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))
    return 0


def other_config_rows(steps: int, timeout_s: int = 900):
    """BASELINE.json's other configurations and the all-double mode, beside the headline: north_star's acceptance is
    stated "on all five configs".  Each row is a short default-arm run of THIS script in a process of its own (so a
    failure or a time-out there can never cost the headline line), with the CPU-oracle leg, the SURVEY 8(f) rows and this
    very step switched off.  Config 1 (7e4 segments, launch-bound: SURVEY.md 8(d) "not meaningful") is a parity case only."""
    import subprocess

    rows = {}
    for key, extra in (("config2", ["--config", "2"]), ("config5", ["--config", "5"]), ("config4", ["--config", "4"]),
                       ("config3_double", ["--config", "3", "--double"])):
        cmd = [sys.executable, os.path.abspath(__file__), "--gpus", "1", "--steps", str(steps), "--warmup", "3",
               "--no-cpu-baseline", "--no-next", "--no-other"] + extra
        t0 = time.perf_counter()
        try:
            env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout_s, env=env)
            line = next((ln for ln in reversed(r.stdout.splitlines()) if ln.startswith("{")), None)
            if r.returncode != 0 or line is None:
                rows[key] = {"error": f"rc={r.returncode}: {(r.stderr or r.stdout)[-400:]}"}
                continue
            j = json.loads(line)
            rf, e2e = j.get("roofline") or {}, j.get("e2e") or {}
            rows[key] = {
                "workload": j["config"]["workload"], "precision": j["config"]["precision"], "value": j["value"], "unit": j["unit"],
                "rays_per_sec": j["rays_per_sec"], "ms_per_step": j["ms_per_step"], "steps": j["steps"],
                "rays_per_step": j["config"]["rays_per_step_per_gpu"], "segments_per_step": j["config"]["segments_per_step_per_gpu"],
                "distinct_batches_cycled": j["config"]["distinct_batches_cycled"],
                "cell_record_path": j["config"]["cell_record_path"], "deferred_tally": j["config"]["deferred_tally"],
                "roofline": {k: rf.get(k) for k in ("frac", "kernel", "kernel_ms", "whole_step_frac", "achieved", "peak", "unit",
                                                    "algorithmic_bytes_per_launch", "frac_of_red_ceiling")},
                "e2e": {k: e2e.get(k) for k in ("value", "ms_per_step", "h2d_bytes_per_step", "d2h_bytes_per_step")},
                "gpu_launches": j.get("gpu_launches"), "clocks": j.get("clocks"),
                "wall_s": round(time.perf_counter() - t0, 1), "command": " ".join(["python", "bench.py"] + cmd[2:]),
            }
        except Exception as e:  # noqa: BLE001 -- a context row must not lose the headline line
            rows[key] = {"error": repr(e), "wall_s": round(time.perf_counter() - t0, 1)}
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="1-based index into BASELINE.json configs (default 3 = PWR)")
    ap.add_argument("--rays", type=int, default=0, help="rays per batch (default: the config's full batch)")
    ap.add_argument("--ref-rays", type=int, default=200_000, help="rays per step of the CPU reference arm")
    ap.add_argument("--cpu-sample-rays", type=int, default=1_000_000, help="rays of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--double", action="store_true", help="all-double mode (MR_PRECISION_DOUBLE, 64-byte ray records): a context line, "
                    "not the headline; the roofline then uses B_seg = 16 + 9K, B_ray = 64 + 32M (SURVEY.md 8(d)); implies --no-next")
    ap.add_argument("--no-next", action="store_true", help="skip the SURVEY 8(f) rows (next-event cast, batch-moment fold)")
    ap.add_argument("--microbench", default="", choices=["", "red"], help="run a micro-benchmark alone and exit")
    ap.add_argument("--no-other", action="store_true", help="skip the other_configs rows (configs 2, 5, 4 and config 3 all-double, each a short "
                                                            "run of this script in a process of its own)")
    ap.add_argument("--other-steps", type=int, default=5, help="timed steps of each other_configs row")
    ap.add_argument("--no-plain", action="store_true", help="skip the second roofline with the dictionary / tiled-index path off")
    ap.add_argument("--batches", type=int, default=0, help="distinct ray batches cycled through (default: 1; config 4: 8 of its 100)")
    ap.add_argument("--ne-rays", type=int, default=2_000_000, help="events per next-event step")
    ap.add_argument("--ne-detectors", type=int, default=4)
    ap.add_argument("--producers", type=int, default=8, help="host threads feeding the producer ring")
    ap.add_argument("--ring-slots", type=int, default=4)
    ap.add_argument("--push-rays", type=int, default=8192, help="rays per mr_ring_push call of a producer (a burst of collision events)")
    ap.add_argument("--ring-slot-rays", type=int, default=1 << 20)
    ap.add_argument("--block-threads", type=int, default=0)
    ap.add_argument("--sort", type=int, default=-1, help="override MR_OPT_SORT_RAYS (default: library default)")
    ap.add_argument("--opt", action="append", default=[], help="library option as ID=VALUE (MR_OPT_* of include/monteray.h), repeatable")
    ap.add_argument("--pre-opt", action="append", default=[], help="like --opt, but set BEFORE the problem is loaded (options read by mr_load_materials)")
    ap.add_argument("--stage-rays", type=int, default=0, help="override MR_OPT_STAGE_RAYS (rays per H2D chunk of a host batch)")
    args = ap.parse_args()
    prob_kw = {}

    if args.impl == "reference":
        return run_reference(args, prob_kw)
    if args.microbench:
        return run_microbench(args)

    import numpy as np
    import torch

    from paper_1706_07476_b200 import MR_OPT_BLOCK_THREADS, MR_OPT_SORT_RAYS, MR_OPT_STAGE_RAYS, MonteRay, multi
    from workloads import CONFIG_NAMES, FULL_RAYS, make_problem, make_rays

    rank, local_rank, world = multi.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        multi.init_process_group("nccl")
    n_rays = args.rays or FULL_RAYS[args.config]

    # all-double mode: genuinely double inputs (nothing rounded to fp32), as tests/test_gpu_double_inputs.py checks
    prob = make_problem(args.config, double_inputs=args.double, **prob_kw)
    # distinct batches cycled through step by step (BASELINE.json config 4: "10^8 rays in 10^6-ray batches"; every
    # rank its own batches: weak scaling)
    nb = args.batches or (8 if args.config == 4 else 1)
    dtype = np.float64 if args.double else np.float32
    batches = [make_rays(prob, n_rays, batch=rank * nb + b, dtype=dtype) for b in range(nb)]
    rays = batches[0]
    if args.double:
        args.no_next = True
    m = MonteRay(local_rank, 1 if args.double else 0)
    for kv in args.pre_opt:
        k, v = kv.split("=")
        m.set_option(int(k), int(v))
    m.load_problem(prob)
    if args.block_threads:
        m.set_option(MR_OPT_BLOCK_THREADS, args.block_threads)
    if args.sort >= 0:
        m.set_option(MR_OPT_SORT_RAYS, args.sort)
    if args.stage_rays:
        m.set_option(MR_OPT_STAGE_RAYS, args.stage_rays)
    for kv in args.opt:
        k, v = kv.split("=")
        m.set_option(int(k), int(v))
    d_batches = [torch.from_numpy(b).to(dev) for b in batches]
    d_rays = d_batches[0]
    h_rays = torch.from_numpy(rays).pin_memory()
    record_path = m.record_path()
    from paper_1706_07476_b200 import (MR_INFO_COARSE_SHIFT, MR_INFO_DEFERRED, MR_INFO_DISTINCT_RECORDS, MR_OPT_TILED_INDEX,
                                       microbench_red)
    deferred = bool(m.get_option(MR_INFO_DEFERRED))
    h_tally = torch.empty(prob.ncell, dtype=torch.float64).pin_memory()
    sampler = ClockSampler(local_rank) if rank == 0 else None

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    # ---------------------------------------------------------------- device-resident steps (value)
    for i in range(max(args.warmup, 3)):
        m.cast_rays(d_batches[i % nb])
    barrier()
    st0 = m.get_stats()
    if sampler:
        sampler.active = True
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for i in range(args.steps):
        m.cast_rays(d_batches[i % nb])
    e1.record()
    barrier()
    if sampler:
        sampler.active = False
    ms_total = multi.max_over_ranks(e0.elapsed_time(e1), dev)
    st1 = m.get_stats()
    seg_step = (st1.segments - st0.segments) // args.steps          # mean over the batches of the timed steps
    launches = st1.kernel_launches - st0.kernel_launches
    seg_all = multi.sum_over_ranks(seg_step, dev)
    value = seg_all * args.steps / (ms_total * 1e-3)
    rays_all = n_rays * world

    # ---------------------------------------------------------------- dominant-kernel time (roofline)
    peak, peak_src = measured_peak()
    dense = prob.config == 5
    workload = CONFIG_NAMES[args.config]

    def kernel_roofline(kernel_name):
        """Algorithmic bytes of the launches just timed over the cast kernel's own CUDA-event time (the library records
        events around every cast-kernel launch on the launching stream; the ordering pre-pass is NOT inside them)."""
        kms, segs = [], []
        for i in range(min(args.steps, 10)):
            s0 = m.get_stats().segments
            m.cast_rays(d_batches[i % nb])
            st = m.get_stats()
            kms.append(st.last_kernel_ms)
            segs.append(st.segments - s0)
        kernel_ms, seg_launch = statistics.mean(kms), statistics.mean(segs)
        alg = algorithmic_bytes(prob, seg_launch, n_rays, dense)
        if args.double:
            alg = seg_launch * (16 + 9 * prob.K) + n_rays * (64 + 32 * prob.M)
        achieved = alg / (kernel_ms * 1e-3) / 1e9
        wl_key = workload + ("_double" if args.double else "")
        if "+" in kernel_name:      # the deferred tally is two kernels per cast: traffic is their sum, the limiter phase A's
            parts = [committed_profile(wl_key, k) for k in kernel_name.split("+")]
            traffic = sum(t for t, _ in parts) if all(t is not None for t, _ in parts) else None
            limiter = {k: l for k, (_, l) in zip(kernel_name.split("+"), parts)} if any(l for _, l in parts) else None
        else:
            traffic, limiter = committed_profile(wl_key, kernel_name)
        return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "achieved_is": "algorithmic bytes (SURVEY.md 8(d)) / cast-kernel time; not DRAM traffic",
                "peak_source": peak_src, "kernel": kernel_name, "kernel_ms": kernel_ms,
                "kernel_ms_excludes": "the ray-ordering pre-pass (5 small kernels per batch); see whole_step_frac",
                "algorithmic_bytes_per_launch": alg, "segments_per_launch": seg_launch,
                "segments_per_sec_at_roofline": peak * 1e9 / (alg / seg_launch),
                "dram_GBps_from_committed_capture": (traffic / (kernel_ms * 1e-3) / 1e9) if traffic else None,
                "limiter": limiter}

    kname = {"coarse_blocks": "cast_defer_kernel+defer_scatter_kernel" if deferred else "cast_kernel<C4>"}.get(
        record_path, f"cast_kernel<{record_path}>")
    roofline = kernel_roofline(kname)
    roofline["whole_step_frac"] = value / world / roofline["segments_per_sec_at_roofline"]
    # the measured L2 fp64-atomic ceiling (one uncoalesced red per lane into an array of the tally's size), same run
    try:
        red = microbench_red(local_rank, prob.ncell, 1, 0, 1 << 27, 3)
        gat = microbench_red(local_rank, prob.ncell, 1, 16, 1 << 27, 3)
        kernel_red_rate = roofline["segments_per_launch"] / (roofline["kernel_ms"] * 1e-3)
        roofline["atomic_ceiling"] = {
            "red_per_sec": red["lane_ops_per_sec"], "red_plus_16B_gather_per_sec": gat["lane_ops_per_sec"],
            "kernel_red_per_sec": kernel_red_rate, "frac_of_red_ceiling": kernel_red_rate / red["lane_ops_per_sec"],
            "how": "mr_microbench_red: random red.global.add.f64 into ncell doubles, 2^27 lane-ops, best of 3"}
    except Exception as e:  # noqa: BLE001
        roofline["atomic_ceiling"] = {"error": repr(e)}
    roofline_plain = None
    if record_path.startswith("tiled") and not args.no_plain:
        m.set_option(MR_OPT_TILED_INDEX, 0)
        plain_path = m.record_path()
        for _ in range(3):
            m.cast_rays(d_rays)
        roofline_plain = kernel_roofline(f"cast_kernel<{plain_path}>")
        roofline_plain["cell_record_path"] = plain_path
        roofline_plain["why"] = ("the headline runs the dictionary + tiled-index path (this mesh has "
                                 f"{m.get_option(MR_INFO_DISTINCT_RECORDS)} distinct cell records); a mesh with more than 1024 "
                                 "distinct records gets this path")
        m.set_option(MR_OPT_TILED_INDEX, 1)

    # the two qualifiers of the headline fraction, inside `roofline` where the driver's parser keeps them
    roofline["frac_of_red_ceiling"] = (roofline.get("atomic_ceiling") or {}).get("frac_of_red_ceiling")
    roofline["plain_records_frac"] = roofline_plain["frac"] if roofline_plain else None
    roofline["plain_records_kernel_ms"] = roofline_plain["kernel_ms"] if roofline_plain else None

    # ---------------------------------------------------------------- end to end through the C ABI, host buffers
    e2e = None
    if not args.no_e2e:
        for _ in range(2):
            m.cast_rays(h_rays)
            m.read_tally_into(h_tally.data_ptr())
        barrier()
        if sampler:
            sampler.active = True
        s_e0 = m.get_stats().segments
        t0 = time.perf_counter()
        for _ in range(args.steps):
            m.cast_rays(h_rays)                    # H2D of the batch from pinned memory, inside the call
            m.read_tally_into(h_tally.data_ptr())  # D2H of the ncell doubles (synchronises)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if sampler:
            sampler.active = False
        dt = multi.max_over_ranks(dt, dev)
        seg_e2e = multi.sum_over_ranks(m.get_stats().segments - s_e0, dev)
        blocking = {"value": seg_e2e / dt, "unit": UNIT, "ms_per_step": 1e3 * dt / args.steps,
                    "read": "mr_read_tally after every batch (blocks until the batch is cast, then copies)"}
        # The same loop with the read-back taken off the critical path: mr_read_tally_async snapshots the tally on the device in
        # stream order and copies the snapshot out on its own stream while the NEXT batch is staged and cast; every step's
        # tally still reaches the host (two alternating page-locked buffers), all transfers end inside the timed region.
        h_tally2 = torch.empty(prob.ncell, dtype=torch.float64).pin_memory()
        bufs = (h_tally, h_tally2)
        for i in range(2):
            m.cast_rays(h_rays)
            m.read_tally_async_into(bufs[i % 2].data_ptr())
        m.sync()
        barrier()
        if sampler:
            sampler.active = True
        s_e0 = m.get_stats().segments
        t0 = time.perf_counter()
        for i in range(args.steps):
            m.cast_rays(h_rays)
            m.read_tally_async_into(bufs[i % 2].data_ptr())
        m.sync()                                       # every queued cast and every read-back has finished
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if sampler:
            sampler.active = False
        dt = multi.max_over_ranks(dt, dev)
        seg_e2e = multi.sum_over_ranks(m.get_stats().segments - s_e0, dev)
        e2e = {"value": seg_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": int(rays.nbytes),
               "d2h_bytes_per_step": int(prob.ncell * 8), "ms_per_step": 1e3 * dt / args.steps,
               "read": "mr_read_tally_async after every batch (device snapshot in stream order, D2H on its own stream, overlapping "
                       "the next batch; two alternating page-locked host buffers; mr_sync before the clock stops)",
               "blocking_read": blocking}
    # ---------------------------------------------------------------- next-event cast, batch-moment fold
    next_rows = None
    if not args.no_next and world == 1:   # context rows, single GPU only; never allowed to cost the headline line
        next_rows = {}
        try:
            lo = np.array([prob.xe[0], prob.ye[0], prob.ze[0]])
            hi = np.array([prob.xe[-1], prob.ye[-1], prob.ze[-1]])
            g = np.random.default_rng(7)
            dets = lo + (0.05 + 0.9 * g.random((args.ne_detectors, 3))) * (hi - lo)   # detector points inside the mesh
            n_ne = min(args.ne_rays, n_rays)
            m.load_detectors(dets)
            d_ev = d_rays[:n_ne]
            for _ in range(3):
                m.cast_next_event(d_ev)
            barrier()
            s0 = m.get_stats()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = max(3, min(args.steps, 10))
            a0.record()
            for _ in range(reps):
                m.cast_next_event(d_ev)
            a1.record()
            barrier()
            ms = a0.elapsed_time(a1) / reps
            s1 = m.get_stats()
            ne_seg = (s1.ne_segments - s0.ne_segments) // reps
            ne_bytes = ne_seg * (4 if dense else 5) * prob.K + n_ne * args.ne_detectors * (32 + 16 * prob.M)
            next_rows["next_event"] = {
                "value": ne_seg / (ms * 1e-3), "unit": "segments/s", "pairs_per_sec": n_ne * args.ne_detectors / (ms * 1e-3),
                "ms_per_step": ms, "events": n_ne, "detectors": args.ne_detectors, "segments_per_step": int(ne_seg),
                "roofline": {"bound": "hbm", "achieved": ne_bytes / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                             "frac": ne_bytes / (ms * 1e-3) / 1e9 / peak,
                             "traffic": committed_profile(workload, "next_event_kernel")[0] if (n_ne, args.ne_detectors) == (2_000_000, 4) else None,
                             "limiter": committed_profile(workload, "next_event_kernel")[1],
                             "algorithmic_bytes": "5K (4K dense) per segment + (32 + 16 M) per (event, detector) pair"}}
            for _ in range(3):
                m.end_batch()
            barrier()
            a0.record()
            for _ in range(reps):
                m.end_batch()
            a1.record()
            barrier()
            ms = a0.elapsed_time(a1) / reps
            fold_bytes = prob.ncell * 40
            next_rows["end_batch"] = {
                "value": prob.ncell / (ms * 1e-3), "unit": "cells/s", "ms_per_step": ms,
                "roofline": {"bound": "hbm", "achieved": fold_bytes / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                             "frac": fold_bytes / (ms * 1e-3) / 1e9 / peak,
                             "algorithmic_bytes": "40 per cell (read tally, read+write previous total and sum of squares)"}}
            # NEXT-1 (Fig. 4): P producer threads push the batch piecewise into the producer ring; buffers ship as they fill.
            # The producers are C threads inside the library (mr_ring_bench_producers): Python threads slicing NumPy arrays
            # measure the interpreter, not the ring
            P = max(1, args.producers)
            piece = max(1, args.push_rays)    # rays per push: a burst of collision events
            slot_rays = min(args.ring_slot_rays, max(1024, n_rays))

            h_ring = (h_tally, torch.empty(prob.ncell, dtype=torch.float64).pin_memory())

            def ring_step(i):
                push_ms = m.ring_bench_producers(rays, P, piece)
                m.read_tally_async_into(h_ring[i % 2].data_ptr())   # every step's tally goes to the host, off the producers' path
                return push_ms

            m.ring_open(args.ring_slots, slot_rays)
            ring_step(0)
            m.sync()
            w0 = m.ring_stats()["producer_wait_ms"]
            casts0, slots0 = m.ring_stats()["casts"], m.ring_stats()["slots_shipped"]
            barrier()
            reps = max(2, min(args.steps, 5))
            t0 = time.perf_counter()
            push_ms = [ring_step(i) for i in range(reps)]
            m.sync()
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) / reps
            rs = m.ring_stats()
            m.ring_close()
            producer_ms = min(m.ring_bench_producers(rays, P, piece, dry_run=True) for _ in range(3))
            device_ms = ms_total / args.steps
            ring_ms = 1e3 * dt
            lo_ms, hi_ms = min(producer_ms, device_ms), max(producer_ms, device_ms)
            next_rows["producer_ring"] = {
                "value": seg_step / dt, "unit": UNIT, "ms_per_step": ring_ms, "producers": P, "rays_per_push": piece,
                "producer_kind": "C threads inside the library (mr_ring_bench_producers)",
                "slots": args.ring_slots, "rays_per_slot": slot_rays,
                # MR_OPT_RING_MERGE (auto): buffers shipped while an earlier cast still runs are cast together, in one launch
                "buffers_shipped_per_step": (rs["slots_shipped"] - slots0) / reps, "casts_per_step": (rs["casts"] - casts0) / reps,
                "rays_per_cast": n_rays * reps / max(1, rs["casts"] - casts0),
                "push_and_flush_ms_per_step": statistics.mean(push_ms),
                "producer_wait_ms_per_step": (rs["producer_wait_ms"] - w0) / reps,
                "producers_alone_ms_per_step": producer_ms,
                "device_only_ms_per_step": device_ms,
                "tally_readback_in_step": "mr_read_tally_async after every step (two alternating page-locked buffers), mr_sync before the clock stops",
                # 1 = the shorter of (producers, device) is hidden completely behind the longer one; 0 = they run back to back
                "overlap": 1.0 - (ring_ms - hi_ms) / lo_ms if lo_ms > 0 else None,
                "overlap_is": "1 - (ring step - max(producers alone, device only)) / min(producers alone, device only); the ring step "
                              "also reads the tally back (D2H of ncell doubles) and casts in several launches (casts_per_step), which neither reference time contains",
                "h2d_bytes_per_step": int(rays.nbytes), "d2h_bytes_per_step": int(prob.ncell * 8)}
            # NEXT-4: the same estimator on an R-Z (cylindrical) pin-cell mesh, its own context
            from workloads import make_rz_problem, make_rz_rays

            rzp = make_rz_problem(256, 2048)
            rz_rays = torch.from_numpy(make_rz_rays(rzp, 4_000_000)).to(dev)
            with MonteRay(local_rank, 0) as mz:
                mz.load_problem(rzp)
                for _ in range(3):
                    mz.cast_rays(rz_rays)
                barrier()
                z0 = mz.get_stats()
                a0.record()
                for _ in range(reps):
                    mz.cast_rays(rz_rays)
                a1.record()
                barrier()
                ms = a0.elapsed_time(a1) / reps
                rz_seg = (mz.get_stats().segments - z0.segments) // reps
            rz_bytes = rz_seg * (16 + 5 * rzp.K) + rz_rays.shape[0] * (32 + 16 * rzp.M)
            next_rows["rz_cast"] = {
                "value": rz_seg / (ms * 1e-3), "unit": UNIT, "rays_per_sec": rz_rays.shape[0] / (ms * 1e-3), "ms_per_step": ms,
                "workload": rzp.name, "rays": int(rz_rays.shape[0]), "segments_per_step": int(rz_seg),
                "roofline": {"bound": "hbm", "achieved": rz_bytes / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                             "frac": rz_bytes / (ms * 1e-3) / 1e9 / peak,
                             "traffic": committed_profile(rzp.name, "rz_kernel")[0],
                             "limiter": committed_profile(rzp.name, "rz_kernel")[1]}}
        except Exception as e:  # noqa: BLE001 -- report, do not lose the JSON line
            next_rows["error"] = repr(e)
    total_launches = m.get_stats().kernel_launches
    m_info = {"distinct": m.get_option(MR_INFO_DISTINCT_RECORDS), "coarse_shift": m.get_option(MR_INFO_COARSE_SHIFT)}
    # replicas are combined by ONE fp64 sum all-reduce of the tally when it is read: timed here, outside `value`
    allreduce_ms = None
    if world > 1:
        t = m.tally_tensor()
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        multi.allreduce_sum_(t)
        a1.record()
        barrier()
        allreduce_ms = multi.max_over_ranks(a0.elapsed_time(a1), dev)

    # ---------------------------------------------------------------- CPU oracle beside it (rank 0, N = 1)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle.vrc_oracle import max_threads

        threads = max(1, min(max_threads(), len(os.sched_getaffinity(0))))
        n_s = min(args.cpu_sample_rays, n_rays)
        rate, segs, dt, used = cpu_oracle_rate(prob, rays[:n_s], threads)
        n_1 = max(1000, n_s // 10)                  # the oracle on ONE thread beside the all-cores figure
        rate1, segs1, dt1, _ = cpu_oracle_rate(prob, rays[:n_1], 1)
        cpu = {"value": rate, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"first {n_s} rays of the batch ({segs} segments), {dt:.1f} s wall on {used} threads",
               "single_thread": {"value": rate1, "unit": UNIT, "sample": f"first {n_1} rays ({segs1} segments), {dt1:.1f} s wall"}}

    other = None
    if rank == 0 and world == 1 and not args.no_other and args.config == 3 and not args.double and not args.rays:
        torch.cuda.synchronize()
        other = other_config_rows(args.other_steps)

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 (everything)" if args.double else "mixed: fp32 tables/rays/coefficients, fp64 walk/score/tally", "data": "synthetic",
            "config": {"workload": CONFIG_NAMES[args.config], "mesh": [prob.nx, prob.ny, prob.nz], "K": prob.K, "M": prob.M,
                       "rays_per_step_per_gpu": n_rays, "segments_per_step_per_gpu": int(seg_step),
                       "precision": "double (everything fp64)" if args.double else "mixed (fp32 tables/rays/coefficients, fp64 walk/score/tally)",
                       "cell_record_path": record_path, "deferred_tally": deferred,
                       "distinct_cell_records": m_info["distinct"], "coarse_block_shift": m_info["coarse_shift"],
                       "distinct_batches_cycled": nb,
                       "parallelism": f"replicas x{world}" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2 (rays 320 MB + cell records 139 MB + tally 69 MB), no flush"
                       if args.config == 3 else "no flush"},
            "rays_per_sec": rays_all * args.steps / (ms_total * 1e-3),
            "roofline": roofline, "roofline_plain_records": roofline_plain, "cpu_baseline": cpu, "e2e": e2e, "next_rows": next_rows,
            "other_configs": other,
            "traffic_is": "dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures "
                          "(profiles/traffic.txt), not measured by this run",
            "traffic_sources": TRAFFIC_SOURCES,
            "allreduce_ms": allreduce_ms,
            "gpu_launches": int(launches), "gpu_launches_total": int(total_launches),
            "clocks": sampler.report() if sampler else None,
        }
        print(json.dumps(out))
    m.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
