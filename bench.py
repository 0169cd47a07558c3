#!/usr/bin/env python
"""Benchmark of the direct-dedispersion hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

A step = one pass of the whole hot path (delay table already in the plan; staging, unpack,
accumulation, store — one dd_execute) over one synthetic filterbank of BASELINE.json's
configs[1] (uint8, 1024 channels x 1024 DM trials x 2^17 samples) resident in HBM.  Prints ONE
JSON line.  `--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same
workload instead.  Under torchrun every rank dedisperses its own beam (independent seeds, no
data-path collective): weak scaling.
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
sys.path.insert(0, ROOT)

from paper_1401_8258_b200 import sharding, synth  # noqa: E402

METRIC = "dedispersed DM·channel·samples/s"
UNIT = "G/s"
SM_COUNT, LANES_PER_SM = 148, 128          # FP32/INT32 add lanes per SM


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.005)

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def visible_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except (ValueError, IndexError):
            pass
    return local_rank


# ----------------------------------------------------------------------------- CPU oracle legs

def oracle_sample(w, seconds_target=12.0):
    """Times oracle/ (as it stands) on a bounded sample of workload w: a subset of DM rows over a
    shortened time range of the same filterbank.  Returns (G/s, cores, description)."""
    import oracle
    cores = oracle.num_threads()
    ms = oracle.max_shift(w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    nsamp = min(w.nsamp, 1 << 15)
    X = synth.make_input(w, nsamp + ms)
    nrows = max(cores, 8)
    rows = np.unique(np.linspace(0, w.ndm - 1, nrows).astype(np.int32))
    f = oracle.dedisperse_f32 if w.dtype == "f32" else oracle.dedisperse_u8
    f(X, 256, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows[:cores])           # warm caches / threads
    t0 = time.perf_counter()
    f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    dt = time.perf_counter() - t0
    # grow the sample towards the time target (once), keeping the run bounded
    grow = int(min(8, seconds_target / max(dt, 1e-3)))
    if grow >= 2:
        rows = np.unique(np.linspace(0, w.ndm - 1, nrows * grow).astype(np.int32))
        t0 = time.perf_counter()
        f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
        dt = time.perf_counter() - t0
    adds = len(rows) * w.nchans * nsamp
    desc = "%d of %d DM rows x %d of %d samples x %d channels, literal (d,t,c) nest" % (
        len(rows), w.ndm, nsamp, w.nsamp, w.nchans)
    return adds / dt / 1e9, cores, desc, dt, (X, nsamp, rows)


def run_reference(args, w):
    rank = _env_int("RANK", 0)
    if rank != 0:
        return
    import oracle
    gps, cores, desc, dt, (X, nsamp, rows) = oracle_sample(w, seconds_target=6.0)
    f = oracle.dedisperse_f32 if w.dtype == "f32" else oracle.dedisperse_u8
    steps = max(1, min(args.steps, 5))
    for _ in range(min(args.warmup, 1)):
        f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    t0 = time.perf_counter()
    for _ in range(steps):
        f(X, nsamp, w.fch1, w.foff, w.tsamp, w.dm_list, rows=rows)
    dt = (time.perf_counter() - t0) / steps
    val = len(rows) * w.nchans * nsamp / dt / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "sample": desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ----------------------------------------------------------------------------- GPU leg

def run_ours(args, w):
    import torch
    import paper_1401_8258_b200 as dd

    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    dtype = dd.DD_F32 if w.dtype == "f32" else dd.DD_U8
    tdt = torch.float32 if w.dtype == "f32" else torch.uint8
    odt = torch.float32 if w.dtype == "f32" else torch.int32
    plan = dd.Plan(dtype, w.nchans, w.fch1, w.foff, w.tsamp, w.dm_list)
    if args.kernel:
        plan.set_kernel({"generic": dd.DD_KERNEL_GENERIC, "tma": dd.DD_KERNEL_TMA, "ps": dd.DD_KERNEL_PS}[args.kernel])
    ms = plan.max_shift()
    nb = w.nbeams
    in_stride = (w.nsamp + ms + 63) // 64 * 64
    out_stride = w.nsamp

    # host input: pinned, one beam per rank-beam (rank r uses beam seeds r*nb .. r*nb+nb-1)
    Xh = torch.empty((nb, w.nchans, in_stride), dtype=tdt).pin_memory()
    Xh.zero_()
    wb = synth.scaled(w, nbeams=max(2, nb * world))           # per-beam seeds
    for b, beam in enumerate(sharding.beams_of_rank(rank, world, nb)):
        Xh[b, :, :w.nsamp + ms] = torch.from_numpy(synth.make_input(wb, w.nsamp + ms, beam=beam))
    Xd = Xh.cuda()
    Dd = torch.empty((nb, w.ndm, out_stride), dtype=odt, device="cuda")
    stream = torch.cuda.Stream()
    kern = plan.kernel_for(Xd, in_stride, w.nchans * in_stride, Dd, out_stride, w.ndm * out_stride, w.nsamp, nb)

    lpe = plan.launches_per_execute()          # kernels per dd_execute (front end + main kernel)
    streamer = None
    if w.nchunks > 1:
        # config 5: fed through the streaming API: first push nsamp/nchunks + maxshift, then equal chunks
        chunk = w.nsamp // w.nchunks
        streamer = dd.Stream(plan, chunk + ms, nb)

    def step():
        if streamer is None:
            plan.execute(Xd, in_stride, w.nchans * in_stride, Dd, out_stride, w.ndm * out_stride,
                         w.nsamp, nb, stream)
            return lpe
        streamer.reset()
        pos = emitted = 0
        chunk = w.nsamp // w.nchunks
        for k in range(w.nchunks):
            n_new = chunk + (ms if k == 0 else 0)
            n = streamer.push(Xd[:, :, pos:], in_stride, w.nchans * in_stride, n_new,
                              Dd[:, :, emitted:], out_stride, w.ndm * out_stride, stream)
            pos += n_new
            emitted += n
        assert emitted == w.nsamp
        return w.nchunks * lpe

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    launches = 0
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            step()
    barrier()
    sampler = ClockSampler(visible_gpu_index(local))
    sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with torch.cuda.stream(stream):
        ev[0].record(stream)
        for i in range(args.steps):
            launches += step()
            ev[i + 1].record(stream)
    barrier()
    clocks = sampler.result()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_step = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = sharding.max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / args.steps
    adds_rank = w.adds
    value = sharding.whole_job_rate(adds_rank, world, ms_per_step * 1e-3) / 1e9

    # ---- end to end through the host-buffer C-ABI call (pinned host X and D; copies inside)
    e2e = None
    if nb == 1 and streamer is None:
        Dh = torch.empty((w.ndm, out_stride), dtype=odt).pin_memory()
        plan.execute_host(Xh[0], in_stride, Dh, out_stride, w.nsamp)          # warm-up (allocates workspace)
        plan.execute_host(Xh[0], in_stride, Dh, out_stride, w.nsamp)
        n_e2e = max(3, min(args.steps, 10))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            plan.execute_host(Xh[0], in_stride, Dh, out_stride, w.nsamp)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = sharding.max_over_ranks(dt, dist, "cuda")
        es = 4 if w.dtype == "f32" else 1
        e2e = {"value": sharding.whole_job_rate(adds_rank, world, dt) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": int(w.nchans * (w.nsamp + ms) * es),
               "d2h_bytes_per_step": int(w.ndm * w.nsamp * 4), "ms_per_step": dt * 1e3,
               "timer": "host wall clock around the synchronous dd_execute_host call, pinned buffers"}
        # the host path must give the same bits as the resident path
        same = bool(torch.equal(Dh[:, :w.nsamp].cuda(), Dd[0][:, :w.nsamp]))
        e2e["matches_resident_result"] = same

    if rank == 0:
        peak_max = SM_COUNT * LANES_PER_SM * (clocks["sm_max_mhz"] or 1965) * 1e6 / 1e12
        kernel_ms = float(np.mean(per_step))
        achieved = adds_rank / (kernel_ms * 1e-3) / 1e12
        hbm_bytes = nb * (w.nchans * (w.nsamp + ms) * (4 if w.dtype == "f32" else 1) + w.ndm * w.nsamp * 4)
        hbm_peak = None
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs")
        except (OSError, ValueError):
            pass
        traffic = None
        try:
            for ln in open(os.path.join(ROOT, "profiles", "dram_traffic.txt")):
                f = ln.split()
                if len(f) >= 3 and not ln.startswith("#") and f[0] == w.name and f[1] == str(kern):
                    traffic = float(f[2])
        except OSError:
            pass
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32" if w.dtype == "u8" else "f32",
            "data": "synthetic",
            "config": {"workload": w.name, "nbeams": nb, "nchans": w.nchans, "ndm": w.ndm,
                       "nsamp": w.nsamp, "maxshift": ms, "tsamp": w.tsamp, "fch1": w.fch1, "foff": w.foff,
                       "kernel": {1: "generic", 2: "tma", 3: "ps"}.get(kern, str(kern)),
                       "parallelism": "beam-per-rank" if world > 1 else "single",
                       "l2": "X+D per step = %.0f MB > 126 MB L2 (no flush needed)" % (hbm_bytes / 1e6)},
            "real_time_factor": w.nsamp * w.tsamp / (ms_per_step * 1e-3),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_max, "unit": "Tadd/s",
                         "frac": achieved / peak_max, "traffic": traffic,
                         "peak_note": "148 SM x 128 add lanes x sm_max_mhz (nominal; DESIGN.md)",
                         "kernel_ms": kernel_ms,
                         "frac_at_sampled_clock": (achieved / (SM_COUNT * LANES_PER_SM * clocks["sm_mhz"] * 1e6 / 1e12)
                                                   if clocks["sm_mhz"] else None),
                         "algorithmic_adds_per_launch": adds_rank,
                         "work_note": ("achieved = nbeams*nchans*ndm*nsamp adds (one per DM-channel-sample, SURVEY "
                                       "8(d)) / CUDA-event time of the step; the ps kernels form each output from the "
                                       "same operands but share partial sums of 4-8 channels between trials "
                                       "(DESIGN.md 5.3), so fewer add instructions are issued"),
                         "hbm_algorithmic_bytes": hbm_bytes,
                         "hbm_achieved_gbs": hbm_bytes / (kernel_ms * 1e-3) / 1e9,
                         "hbm_peak_gbs_measured": hbm_peak},
            "clocks": clocks, "gpu_launches": launches,
        }
        if e2e is not None:
            line["e2e"] = e2e
        if not args.no_cpu and world >= 1:
            gps, cores, desc, dt, _ = oracle_sample(w)
            line["cpu_baseline"] = {"value": gps, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": desc, "seconds": dt}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); default 2 = configs[1]")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default=None, choices=["generic", "tma", "ps"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--nsamp", type=int, default=0,
                    help="profiling aid: cut the workload to this many output samples (the line then names it)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = synth.WORKLOADS[args.config]
    if args.nsamp:
        w = synth.scaled(w, nsamp=args.nsamp, name="%s_cut_to_%d_samples" % (w.name, args.nsamp))
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
