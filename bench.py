#!/usr/bin/env python
"""bench.py -- throughput of the dedispersion hot path on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one dd_execute over one seeded synthetic batch: pack/decimate of every DM range
 + tiled dedispersion of every range (a3) + the fp32 DM-time writer (a4).
Workload at N=1: BASELINE.json configs[2], the 4096-channel SPOTLIGHT-shaped beam the north_star's
>=60 % roofline target is quoted on.  N>1: one process per GPU, each dedisperses its own beam of that
shape (beams are independent) -- weak scaling, no collective on the data path.

  value        DM-trial x samples per second, whole job, inputs resident in HBM (CUDA events).
  e2e          the same through dd_execute_host_async (steps queued back to back) + dd_host_wait: pinned host buffers,
               H2D + D2H of every step inside the timed region; the synchronous dd_execute_host figure beside it.
  roofline     dominant kernel (dd_tiled_kernel): brute-force adds / its device time, against the FP32-add
               issue peak SMs x 128 lanes x 1.965 GHz; "bound": "alu".
  cpu_baseline the oracle (oracle/, plain C + OpenMP, as it stands) on a bounded sample, rank 0, N=1.
  --impl reference: the oracle alone on the host cores (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2605_03531_b200 import workloads as W  # noqa: E402

METRIC = "dedispersed DM-trial x samples per second"
UNIT = "DM-trial*samples/s"
WORKLOAD_KEY = 3  # BASELINE.json configs[2]
FP32_LANES_PER_SM = 128
# dram__bytes_read.sum + dram__bytes_write.sum of every dd_tiled_kernel launch of one step, from the committed ncu
# capture (one launch per ncu run, so no counter is lost to multi-pass replay); see the .md beside it for the command
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_dd_tiled_kernel_traffic.csv")


def ncu_traffic_per_launch(workload_name: str):
    """Mean DRAM bytes (read + write) per dd_tiled_kernel launch of `workload_name` from TRAFFIC_CSV, or None."""
    try:
        import csv
        with open(TRAFFIC_CSV) as fh:
            rows = [r for r in csv.DictReader(l for l in fh if not l.startswith("#")) if r["workload"] == workload_name]
        vals = [float(r["dram_read_bytes"]) + float(r["dram_write_bytes"]) for r in rows]
        return sum(vals) / len(vals) if vals else None
    except Exception:
        return None


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, uuid: str | None = None, period_s: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid) if uuid else pynvml.nvmlDeviceGetHandleByIndex(index)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    _NAMES = {
        0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x10: "sync_boost",
        0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
        0x100: "display_clock_setting",
    }

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self._NAMES.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        med = int(statistics.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline and --impl reference): the only places bench.py touches oracle/
# --------------------------------------------------------------------------------------------------
def oracle_sample_run(w, x_beam: np.ndarray, trials_per_range: int):
    """Time the oracle on `trials_per_range` evenly spaced trials of every range of one beam, full valid
    span, decimation included.  Returns (seconds, dm_samples_done, threads, description)."""
    import oracle  # test infrastructure; allowed here (cpu_baseline / reference arm only)

    oracle.build()
    threads = oracle.num_threads()
    done = 0
    t0 = time.perf_counter()
    for rg in w.ranges:
        tab = oracle.delay_table(w.f_top_mhz, w.chan_width_mhz, w.nchans, w.tsamp_s, rg.decim, rg.dm_lo, rg.dm_step, rg.ndm)
        ns_r, maxd, nout = oracle.range_sizes(w.nsamps, rg.decim, tab)
        y = oracle.decimate(x_beam, rg.decim)
        n = min(trials_per_range, rg.ndm)
        sel = np.unique(np.linspace(0, rg.ndm - 1, n).astype(np.int32))
        out = oracle.dedisperse(y, tab, sel=sel, t0=0, nt=nout)
        done += out.shape[0] * out.shape[1]
        del y, out
    dt = time.perf_counter() - t0
    desc = "%d evenly spaced trials of each of the %d ranges, full valid span, %d channels, decimation included" % (
        trials_per_range, len(w.ranges), w.nchans)
    return dt, done, threads, desc


def run_reference(args, w):
    """--impl reference: the oracle as it stands on the host cores; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    x = W.generate_beam(w, 0)
    per_step = []
    for i in range(args.warmup + args.steps):
        dt, done, threads, desc = oracle_sample_run(w, x, args.ref_trials)
        if i >= args.warmup:
            per_step.append((dt, done))
    tot_t = sum(a for a, _ in per_step)
    tot_n = sum(b for _, b in per_step)
    value = tot_n / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, len(per_step)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u%d" % w.in_bits,
        "data": "synthetic", "config": {"workload": w.name, "sample_per_step": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------------------
def aggregate(total_units: float, elapsed_ms_local: float, dist=None, device=None):
    """Whole-job value: units of all ranks / max-over-ranks time.  Works with gloo (CPU) and nccl."""
    import torch

    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([elapsed_ms_local], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        u = torch.tensor([total_units], dtype=torch.float64, device=device)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
        return float(u.item()), float(t.item())
    return float(total_units), float(elapsed_ms_local)


def run_stub(args, w):
    """--stub-body (tests only): the N-rank plumbing of run_ours -- rendezvous, one seeded beam per rank, barrier,
    max-over-ranks time, summed units, rank 0 prints -- over gloo on CPU with the timed GPU body replaced by a
    sleep.  Lets `bench.py --gpus 2` be run as a command where there is no GPU.  Never a bench value."""
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    small = W.scaled(w, nchans=32, nsamps=2048, ranges=[W.DMRange(0.0, 1.0, 4, 1)])
    x = W.generate_beam(small, beam=rank)                      # every rank its own seeded beam
    units_local = 1000.0 * args.steps
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    time.sleep(0.01 * (rank + 1) * args.steps)                 # stands in for the timed dd_execute loop
    ms_local = (time.perf_counter() - t0) * 1e3
    if world > 1:
        dist.barrier()
    units, ms_total = aggregate(units_local, ms_local, dist if world > 1 else None, None)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": units / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps,
                          "stub": True, "units": units, "beam_checksum_rank0": int(x.sum()),
                          "config": {"workload": w.name, "parallelism": "replicas: one beam per GPU, no collective"}}),
              flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def self_launch(args, argv):
    """`python bench.py --gpus N` with N > 1 outside torchrun: start the N ranks ourselves (one process per GPU),
    exactly as the driver would: torch.distributed.run --nnodes=1 --nproc-per-node N on 127.0.0.1."""
    import socket
    import subprocess

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd, env=dict(os.environ, MASTER_ADDR="127.0.0.1"))


def time_config(B, torch, key, steps, warmup, dev, sms, f_max):
    """One line of `other_configs`: ms per dd_execute, DM-samples/s and fraction of the FP32-add roofline of BASELINE
    config `key`, same event timing as the headline.  Kernel timing does not depend on the sample values, so the
    input is seeded random bytes drawn on the device (the parity tests use the real generators)."""
    w = W.CONFIGS[key]
    plan = B.Plan.from_workload(w)
    dm_samples, adds = plan.work()
    g = torch.Generator(device=dev)
    g.manual_seed(w.seed)
    x = torch.randint(0, 256, (w.in_bytes,), dtype=torch.uint8, device=dev, generator=g)
    out = torch.empty(plan.out_elems(), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        plan.execute(x, out, stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(steps):
        plan.execute(x, out, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    tiles = [plan.tile_info(r) for r in range(plan.nranges)]
    res = {"workload": w.name, "ms_per_execute": ms, "dm_samples_per_s": dm_samples / (ms * 1e-3), "adds": adds,
           "frac_of_fp32_add_roofline": adds / (ms * 1e-3) / (sms * FP32_LANES_PER_SM * f_max),
           "input_gb_per_s": w.in_bytes / (ms * 1e-3) / 1e9, "dtype": "u%d" % w.in_bits, "nbeams": w.nbeams,
           "lanes_mode_per_range": [[t["lanes"], t["mode"]] for t in tiles], "steps": steps,
           "input": "seeded random bytes drawn on the device (timing only)"}
    plan.destroy()
    del x, out
    torch.cuda.empty_cache()
    return res


def run_ours(args, w):
    if args.stub_body:
        return run_stub(args, w)
    import torch
    import torch.distributed as dist

    from paper_2605_03531_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # one beam per rank, a different seeded beam each (weak scaling over independent beams)
    x_host = W.generate_beam(w, beam=rank)
    plan = B.Plan.from_workload(w)
    if args.variant:
        plan.set_kernel(args.variant)
    dm_samples, adds = plan.work()
    x = torch.from_numpy(x_host.view(np.int16) if x_host.dtype == np.uint16 else x_host).to(dev)
    out = torch.empty(plan.out_elems(), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    for _ in range(args.warmup):
        plan.execute(x, out, stream)
    torch.cuda.synchronize()
    plan.set_profiling(args.steps)
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local_rank, uuid)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    e0.record(stream)
    for _ in range(args.steps):
        plan.execute(x, out, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    ms_local = e0.elapsed_time(e1)
    units, ms_total = aggregate(dm_samples * args.steps, ms_local, dist if world > 1 else None, dev)
    value = units / (ms_total * 1e-3)

    # dominant kernel: dd_tiled_kernel, timed live by events around each launch inside dd_execute
    tiled_ms, pack_ms, n_tiled = 0.0, 0.0, 0
    for s in range(args.steps):
        for k in plan.kernel_times(s):
            if k["kind"] == "pack":
                pack_ms += k["ms"]
            else:
                tiled_ms += k["ms"]
                n_tiled += 1
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peaks = _measured_peaks()
    f_max = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    peak_adds = sms * FP32_LANES_PER_SM * f_max
    achieved = adds * args.steps / (tiled_ms * 1e-3)
    roofline = {
        "bound": "alu", "achieved": achieved / 1e12, "peak": peak_adds / 1e12, "unit": "Tadd/s",
        "frac": achieved / peak_adds, "traffic": ncu_traffic_per_launch(w.name),
        "traffic_source": "profiles/r2_dd_tiled_kernel_traffic.csv (ncu dram__bytes_read.sum + dram__bytes_write.sum, mean over the launches of one step)",
        "kernel": "dd_tiled_kernel", "launches_timed": n_tiled,
        "adds_per_launch": adds / max(1, n_tiled // max(1, args.steps)),
        "avg_launch_ms": tiled_ms / max(1, n_tiled),
        "kernel_share_of_step": tiled_ms / (ms_local if ms_local > 0 else 1.0),
        "pack_share_of_step": pack_ms / (ms_local if ms_local > 0 else 1.0),
        "peak_source": "SMs x 128 FP32 lanes x sm_max_mhz of MEASURED_PEAKS.json" if peaks else
                       "SMs x 128 FP32 lanes x 1965 MHz (fallback: MEASURED_PEAKS.json absent)",
        "whole_step_frac": (adds * args.steps / (ms_local * 1e-3)) / peak_adds,
        "hbm_frac_of_measured": ((w.nchans * w.nsamps * (w.in_bits // 8) + plan.out_elems() * 4) * args.steps
                                 / (ms_local * 1e-3)) / (float(peaks.get("hbm_gbs", 6650.0)) * 1e9),
    }

    # end to end through the C ABI with host buffers (pinned), H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        hin = torch.from_numpy(x_host.view(np.int16) if x_host.dtype == np.uint16 else x_host).pin_memory()
        # two output buffers used alternately: consecutive steps of the pipelined call may copy back at the same time
        houts = [torch.empty(plan.out_elems(), dtype=torch.float32).pin_memory() for _ in range(2)]
        plan.set_profiling(0)
        for s in range(2):  # allocates both slots of staging buffers, warms up
            plan.execute_host(hin, houts[s], stream)
        n_e2e = max(1, min(args.steps, args.e2e_steps or args.steps))
        # (a) one synchronous call per step: upload, kernels, download (overlapped inside the call), wait
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for s in range(n_e2e):
            plan.execute_host(hin, houts[s % 2], stream)
        torch.cuda.synchronize()
        sync_ms = (time.perf_counter() - t0) * 1e3 / n_e2e
        # (b) the headline: the same steps queued back to back (dd_execute_host_async), one wait at the end; every step
        # still uploads its input and downloads its whole result inside the timed region
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for s in range(n_e2e):
            plan.execute_host_async(hin, houts[s % 2], stream)
        plan.host_wait()
        torch.cuda.synchronize()
        dt_ms = (time.perf_counter() - t0) * 1e3
        u2, ms2 = aggregate(dm_samples * n_e2e, dt_ms, dist if world > 1 else None, dev)
        e2e = {"value": u2 / (ms2 * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(hin.numel() * hin.element_size()),
               "d2h_bytes_per_step": int(houts[0].numel() * 4), "steps": n_e2e, "ms_per_step": ms2 / n_e2e,
               "api": "dd_execute_host_async x steps + dd_host_wait (C ABI, pinned host buffers, two staging slots: the "
                      "upload of step i+1 and the end of the download of step i overlap the kernels in between)",
               "ms_per_step_synchronous_calls": sync_ms,
               "value_synchronous_calls": dm_samples / (sync_ms * 1e-3)}
        del hin, houts

    # NEXT-2: boxcar single-pulse search over the plane just written -- an extra, HBM-bound step
    # reported beside the metric, not inside `value`
    sps = None
    if not args.no_sps and w.in_bits == 8:
        K, thr = 8, 6.0
        rows = plan.sps_rows()
        snr = torch.empty((rows, K), dtype=torch.float32, device=dev)
        tmx = torch.empty((rows, K), dtype=torch.int32, device=dev)
        cnt = torch.empty((rows, K), dtype=torch.int32, device=dev)
        offs = torch.empty(rows * K + 1, dtype=torch.int64, device=dev)
        cand = torch.empty((1 << 20, 4), dtype=torch.int32, device=dev)
        stats = torch.zeros((rows, 2), dtype=torch.int64, device=dev)

        def timed(fn, reps=5):
            for _ in range(2):
                fn()
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            s0.record(stream)
            for _ in range(reps):
                fn()
            s1.record(stream)
            torch.cuda.synchronize()
            return s0.elapsed_time(s1) / reps

        plan.set_profiling(0)
        two_pass_ms = timed(lambda: plan.sps_execute(out, K, thr, snr, tmx, cnt, stream))
        # row statistics from the dedispersion epilogue (dd_plan_set_row_stats): the search then reads the plane once
        plan.set_row_stats(stats)
        exec_stats_ms = timed(lambda: plan.execute(x, out, stream), reps=3)
        sps_ms = timed(lambda: plan.sps_execute(out, K, thr, snr, tmx, cnt, stream))
        cand_ms = timed(lambda: plan.sps_candidates(out, K, thr, cnt, offs, cand, cand.shape[0], stream))
        plan.set_row_stats(None)
        plane_bytes = plan.out_elems() * 4
        hbm = float(peaks.get("hbm_gbs", 6650.0))
        sps = {"kernel": "dd_sps_warp_kernel (one launch for all ranges)", "widths": K, "threshold": thr, "ms": sps_ms, "rows": rows,
               "row_statistics": "from the dedispersion epilogue (dd_plan_set_row_stats): one pass over the plane",
               "ms_two_pass_without_epilogue_statistics": two_pass_ms, "ms_dd_execute_with_statistics": exec_stats_ms,
               "ms_candidate_list": cand_ms, "candidates_above_threshold": int(offs[-1].item()),
               "roofline": {"bound": "hbm", "achieved": plane_bytes / (sps_ms * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                            "frac": plane_bytes / (sps_ms * 1e-3) / 1e9 / hbm,
                            "algorithmic_bytes": "the DM-time plane read once (4 B per DM-trial sample)"}}
        del snr, tmx, cnt, offs, cand, stats

    # NEXT-4: the pulsar-side chain on the rows of range 0 of the plane just written:
    # downsample by 8 -> running-median de-reddening (window 129) -> re-sampling; HBM-bound steps except the median
    post = None
    if rank == 0 and world == 1 and not args.no_post:
        try:
            info = plan.range_info(0)
            ndm, nout, pitch = info["ndm"], info["nout"], info["pitch"]
            src = out[info["offset"]:]
            F, Wn = 8, 129
            nd = nout // F
            hbm = float(peaks.get("hbm_gbs", 6650.0))
            d = torch.empty((ndm, nd), dtype=torch.float32, device=dev)
            rr = torch.empty((ndm, nd), dtype=torch.float32, device=dev)
            rs = B.Resample(1.4, -2.0e-4, 0.0, w.tsamp_s * F, nd)
            rsm = torch.empty((ndm, rs.out_len), dtype=torch.float32, device=dev)

            def timed_post(fn, reps=5):
                fn()
                s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                s0.record(stream)
                for _ in range(reps):
                    fn()
                s1.record(stream)
                torch.cuda.synchronize()
                return s0.elapsed_time(s1) / reps

            t_ds = timed_post(lambda: B.post_downsample(src, ndm, pitch, nout, F, d, nd, stream))
            t_md = timed_post(lambda: B.post_dered(d, ndm, nd, nd, Wn, None, rr, nd, stream))
            t_rs = timed_post(lambda: rs.execute(rr, ndm, nd, rsm, rs.out_len, stream))

            def line(ms, nbytes, bound):
                return {"ms": ms, "bound": bound, "achieved_gb_s": nbytes / (ms * 1e-3) / 1e9,
                        "frac_of_hbm_peak": nbytes / (ms * 1e-3) / 1e9 / hbm}

            post = {"rows": ndm, "samples_per_row": nout, "downsample_factor": F, "median_window": Wn,
                    "downsample": line(t_ds, ndm * (nout + nd) * 4, "hbm"),
                    "running_median": dict(line(t_md, ndm * nd * 8, "alu (order statistics; HBM bytes shown for scale)"),
                                           samples_per_s=ndm * nd / (t_md * 1e-3)),
                    "resample": line(t_rs, ndm * (nd + rs.out_len) * 4, "hbm")}
            rs.destroy()
            del d, rr, rsm
        except Exception as e:
            post = {"skipped": repr(e)}

    # NEXT-3: the exact two-channel sub-band variant, an opt-in shortcut that performs about half the
    # adds of the brute-force count the roofline divides by -- reported beside the metric, never inside `value`
    subband = None
    if rank == 0 and world == 1 and not args.no_subband and not args.variant:
        try:
            plan.set_profiling(0)
            plan.set_kernel(B.DD_KERNEL_SUBBAND)
            for _ in range(2):
                plan.execute(x, out, stream)
            b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            b0.record(stream)
            for _ in range(5):
                plan.execute(x, out, stream)
            b1.record(stream)
            torch.cuda.synchronize()
            sb_ms = b0.elapsed_time(b1) / 5
            executed = plan.executed_adds()
            subband = {"variant": "DD_KERNEL_SUBBAND (exact two-channel sub-bands)", "ms_per_execute": sb_ms,
                       "dm_samples_per_s": dm_samples / (sb_ms * 1e-3), "executed_adds": executed, "brute_force_adds": adds,
                       "executed_over_brute_force": executed / adds,
                       "brute_force_add_bound_ms": adds / peak_adds * 1e3,
                       "ranges_on_pair_rows": [bool(plan.pair_info(r)["enabled"]) for r in range(plan.nranges)],
                       "launches_per_execute": plan.launches(), "workspace_bytes": plan.workspace_bytes()}
            plan.set_kernel(B.DD_KERNEL_AUTO)
        except Exception as e:
            subband = {"skipped": repr(e)}

    # the other BASELINE configs (1, 2, 4, 5), reported beside the headline: `value` stays on config 3
    other = None
    if rank == 0 and world == 1 and not args.no_other_configs:
        del x, out
        torch.cuda.empty_cache()
        other = []
        for key in (1, 2, 4, 5):
            if key == args.workload:
                continue
            try:
                other.append(time_config(B, torch, key, 5 if key != 5 else 3, 3, dev, sms, f_max))
            except Exception as e:  # e.g. a smaller GPU: say so instead of dropping the line
                other.append({"workload": W.CONFIGS[key].name, "skipped": repr(e)})

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        dt, done, threads, desc = oracle_sample_run(w, x_host, args.ref_trials)
        cpu_baseline = {"value": done / dt, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                        "seconds": dt}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u%d" % w.in_bits, "data": "synthetic",
            "config": {"workload": w.name, "nchans": w.nchans, "nsamps": w.nsamps, "beams_per_gpu": 1,
                       "dm_trials": w.total_trials, "ranges": [[r.dm_lo, r.dm_step, r.ndm, r.decim] for r in w.ranges],
                       "l2": "inputs larger than L2 (1.07 GB input, 3.8 GB of packed copies written and read through a 2.2 GB scratch, 3.8 GB output per step)",
                       "parallelism": "replicas: one beam per GPU, no collective"},
            "input_gb_per_s": world * w.nchans * w.nsamps * (w.in_bits // 8) / (ms_total / args.steps * 1e-3) / 1e9,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "sps": sps, "post": post, "subband": subband, "other_configs": other,
            "gpu_launches": plan.launches() * args.steps, "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=WORKLOAD_KEY, help="BASELINE config number (1-5); default 3")
    ap.add_argument("--ref-trials", type=int, default=48, help="oracle sample: trials per range")
    ap.add_argument("--e2e-steps", type=int, default=0, help="end-to-end steps (0 = as many as --steps)")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--no-subband", action="store_true")
    ap.add_argument("--no-post", action="store_true")
    ap.add_argument("--variant", type=int, default=0, help="dd_plan_set_kernel variant of the timed plan (measurements)")
    ap.add_argument("--stub-body", action="store_true", help=argparse.SUPPRESS)  # tests: N-rank plumbing on CPU / gloo
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sps", action="store_true")
    args = ap.parse_args(argv)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        return self_launch(args, sys.argv[1:] if argv is None else argv)
    if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%s" % (args.gpus, os.environ.get("WORLD_SIZE")))
    w = W.CONFIGS[args.workload]
    if w.nbeams > 1:
        w = W.scaled(w, nbeams=1, name=w.name + "_1beam_per_gpu")
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    sys.exit(main())
