#!/usr/bin/env python
"""bench.py -- template-segments/s of the matched-filter + chi^2 hot path on B200.

Contract (driver): `python bench.py --gpus N --steps K --warmup W [--impl reference]` prints ONE JSON line.

  step      = one pass of the whole hot path (a1-a5: template generation, correlate, p band inverse
              FFTs, rho, chi^2, window maxima, trigger compaction + read-back) over the whole bank of
              BASELINE.json:configs[2] (N = 2^20, 1024 templates, p = 16) against one segment.
  value     = template-segments/s with segment, PSD and bank resident in HBM when the timed region starts.
  e2e       = the same through the C ABI with HOST buffers: every step uploads the segment from pinned host memory
              (gwmf_load_segment with the PSD kept: the PSD is loaded once, before the timed region), filters the bank
              and reads the events back; the upload overlaps the previous step's filters on the library's upload stream.
  roofline  = the dominant kernel's algorithmic bytes / its device time (CUDA events recorded by the library on its own
              stream around the stages of every launch, gwmf_filter_timed) against the measured copy bandwidth in
              MEASURED_PEAKS.json.  The path that runs is the library's choice at this size, the decimated path:
              n complex fp32 written by pass 1 and read by pass 2 per n-point transform that is really run (about 1.7
              per template-segment instead of p = 16).  `--path fused` reports the spill-free kernel against the FP32
              ALU peak instead.
  clocks    = SM clock / power / throttle reasons sampled through NVML every 5 ms from the start of the timed region
              to the end of the e2e region.
  cpu_baseline = the fp64 oracle as it stands, on the host cores, on a bounded sample of the workload.
  N > 1     : one process per GPU; every rank filters the whole bank against its own segment (seed +
              rank): independent units, no data-path collective, weak scaling.

`--impl reference` times the oracle (the reference arm of this tier) on the same config and metric.
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
sys.path.insert(0, ROOT)

import workloads as inputs  # noqa: E402

METRIC = "template-segments/sec at N=2^20, p=16 (SNR+chi^2)"
UNIT = "template-segments/s"

# --workload: the default is the headline config (BASELINE.json:configs[2], the one `metric` is quoted on); the
# others are the remaining configs and the "next" rows of SURVEY.md 8(f), measured with the same protocol (their
# lines are records for DESIGN.md, not the contract's metric).
WORKLOADS = {
    "headline": dict(config=2, p=None, templates=None, metric=METRIC,
                     text="BASELINE.json:configs[2]: N=2^20 (256 s at 4096 Hz), 1024 templates (total mass 2-34 Msun, "
                          "grid uniform in eta and chirp mass), p=16, threshold 6, window 4096; Eq. 2 coloured Gaussian "
                          "noise + 10 injections, seed 2 (+rank)"),
    "config1": dict(config=1, p=None, templates=None, metric="template-segments/sec at N=2^18, p=16 (SNR+chi^2)",
                    text="BASELINE.json:configs[1]: N=2^18 (64 s), 256 templates on a grid of m1,m2 in [1,3] Msun, p=16, "
                         "threshold 6, window 4096, 3 injections, seed 1"),
    "config4": dict(config=4, p=None, templates=None, metric="template-segments/sec at N=2^22, p=32 (SNR+chi^2)",
                    text="BASELINE.json:configs[4]: N=2^22 (1024 s), 512 templates with m1,m2 in [1,2] Msun, p=32, "
                         "threshold 5.5, window 4096, 4 injections, seed 4"),
    "snr_only": dict(config=2, p=1, templates=None, metric="template-segments/sec at N=2^20, p=1 (SNR only, PAPER.md:164)",
                     text="SURVEY.md 8(f)-2: configs[2]'s segment and bank with p=1 (one inverse FFT per template, no chi^2)"),
    "sweep": dict(config=3, p=None, templates=None,
                  metric="sustained template-segments/sec over the 15-segment x 4096-template bank sweep at N=2^20, p=16 "
                         "(SNR+chi^2), segment uploads included and overlapped",
                  text="BASELINE.json:configs[3]: 15 half-overlapping segments of N=2^20 from one seeded 2^23-sample stream "
                       "(Eq. 2 noise + 16 injections, seed 3), each against a 4096-template bank (total mass 2-34 Msun), "
                       "p=16, threshold 6, window 4096"),
    "long16": dict(config=4, p=16, templates=None, metric="template-segments/sec at N=2^22, p=16 (SNR+chi^2)",
                   text="SURVEY.md 8(f)-3: configs[4]'s segment (N=2^22, 1024 s) and bank (512 templates, m1,m2 in [1,2] "
                        "Msun) with the headline p=16, threshold 5.5"),
}


def load_workload(name):
    spec = WORKLOADS[name]
    w = inputs.workload(spec["config"], spec["templates"])
    if spec["p"] is not None:
        w.p = spec["p"]
    return w, spec


FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md fallback, only if MEASURED_PEAKS.json is absent


def alu_peak():
    """FP32 non-tensor peak in TFLOP/s: 148 SMs x 128 lanes x 2 flop x max SM clock."""
    mhz, src = 1965.0, "B200 nominal max SM clock"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            mhz, src = float(json.load(fh)["sm_max_mhz"]), "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        pass
    return 148 * 128 * 2 * mhz * 1e6 / 1e12, "148 SMs x 128 FP32 lanes x 2 flop x %.0f MHz (%s)" % (mhz, src)


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def shard_plan(world_size: int, rank: int, n_templates: int, shard: str = "segments"):
    """Returns (segment_seed_offset, first_template, count).
    shard = "segments" (weak scaling, the default): every rank owns the whole bank against its OWN segment (seed offset =
    rank): n_templates template-segments per rank, no data-path communication.
    shard = "templates" (strong scaling, SURVEY.md 8(e) / PAPER.md:196): ONE segment, the bank split into contiguous
    ranges of template ids; the segment is broadcast once, the per-rank event lists are gathered in template order."""
    assert 0 <= rank < world_size
    if shard == "segments":
        return rank, 0, n_templates
    base, rem = divmod(n_templates, world_size)
    first = rank * base + min(rank, rem)
    return 0, first, base + (1 if rank < rem else 0)


def gather_triggers(trig, dist=None, device=None):
    """Template-sharded mode: concatenate the ranks' event lists (each already sorted by (template, window), ranges of
    template ids ascending with the rank) into the bank's list on every rank: an all_gather of fixed-capacity
    buffers, the capacity being the largest per-rank count."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return trig
    import torch
    world = dist.get_world_size()
    dev = device if device is not None else "cpu"
    cnt = torch.tensor([len(trig)], dtype=torch.int64, device=dev)
    counts = [torch.zeros_like(cnt) for _ in range(world)]
    dist.all_gather(counts, cnt)
    cap = max(int(c.item()) for c in counts)
    buf = torch.zeros(max(cap, 1) * 16, dtype=torch.uint8, device=dev)
    raw = torch.from_numpy(np.frombuffer(trig.tobytes(), dtype=np.uint8).copy())
    buf[: raw.numel()] = raw.to(dev)
    bufs = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(bufs, buf)
    parts = [np.frombuffer(b.cpu().numpy().tobytes()[: int(c.item()) * 16], dtype=trig.dtype) for b, c in zip(bufs, counts)]
    return np.concatenate(parts) if parts else trig


def reduce_max_ms(ms: float, dist=None, device=None) -> float:
    """MAX over ranks of a duration (all ranks get the result)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed regions: in-process through NVML every 5 ms (a
    timed region of a few tens of ms still gets >= 10 samples); `nvidia-smi -lms 100` in a child process if NVML
    cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    PERIOD_S = 0.005

    def __init__(self, index: int, uuid: str | None = None):
        self.index = index
        self.uuid = uuid
        self.rows = []                     # (sm_mhz, power_w, reasons bitmask) or nvidia-smi csv rows
        self.proc = None
        self.nvml = None
        self.handle = None
        self.max_mhz = None
        self.stop_flag = threading.Event()
        self.thread = None

    def _nvml_open(self):
        import pynvml
        pynvml.nvmlInit()
        h = None
        if self.uuid:
            for cand in (self.uuid, "GPU-" + self.uuid):
                try:
                    h = pynvml.nvmlDeviceGetHandleByUUID(cand.encode() if isinstance(cand, str) else cand)
                    break
                except Exception:
                    h = None
        if h is None:
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
        self.nvml, self.handle = pynvml, h
        self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))

    def _nvml_loop(self):
        nv, h = self.nvml, self.handle
        reasons_fn = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self.stop_flag.is_set():
            try:
                self.rows.append((float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                  nv.nvmlDeviceGetPowerUsage(h) / 1e3, int(reasons_fn(h))))
            except Exception:
                pass
            self.stop_flag.wait(self.PERIOD_S)

    def start(self):
        try:
            self._nvml_open()
            self.thread = threading.Thread(target=self._nvml_loop, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        if self.nvml is not None:
            self.stop_flag.set()
            self.thread.join(timeout=1)
            nv = self.nvml
            bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
            sm = [r[0] for r in self.rows]
            power = [r[1] for r in self.rows]
            mask = 0
            for r in self.rows:
                mask |= r[2]
            reasons = sorted(nm for nm in names if mask & bits[nm])
            try:
                nv.nvmlShutdown()
            except Exception:
                pass
            return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_min_mhz": float(np.min(sm)) if sm else None,
                    "sm_max_mhz": self.max_mhz, "reasons": reasons, "samples": len(sm),
                    "power_w": float(np.median(power)) if power else None, "sampler": "NVML in-process, every 5 ms"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["NVML and nvidia-smi unavailable"], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], None, set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                power.append(float(r[2]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "power_w": float(np.median(power)) if power else None, "sampler": "nvidia-smi -lms 100"}


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_rate(w, s64, Sn, n_templates: int, threads: int):
    """Template-segments/s of the oracle on `n_templates` templates of the workload (evenly spread over the bank)."""
    import oracle
    idx = np.linspace(0, len(w.masses) - 1, n_templates).astype(int)
    sub = [w.masses[i] for i in idx]
    t0 = time.perf_counter()
    out = oracle.filter_bank(s64, Sn, sub, w.p, w.window, w.rho_thresh, n_threads=threads)
    dt = time.perf_counter() - t0
    assert np.all(out["status"] == 0)
    return n_templates / dt, dt


def base_line(args, w, value, ms_per_step, dtype):
    return {
        "metric": WORKLOADS[args.workload]["metric"], "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": dtype, "data": "synthetic",
        "config": {"workload": WORKLOADS[args.workload]["text"],
                   "n": w.n, "templates": len(w.masses), "p": w.p, "window": w.window,
                   "rho_thresh": w.rho_thresh, "units_per_step": len(w.masses) * args.gpus},
    }


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, _ = load_workload(args.workload)
    s64 = inputs.segment(w).astype(np.float32).astype(np.float64)
    Sn = w.psd
    cores = min(host_cores(), 32)
    per_step = cores                      # one template-segment per thread and step
    for _ in range(args.warmup):
        oracle_rate(w, s64, Sn, per_step, cores)
    t_total = 0.0
    for _ in range(args.steps):
        _, dt = oracle_rate(w, s64, Sn, per_step, cores)
        t_total += dt
    value = per_step * args.steps / t_total
    line = base_line(args, w, value, 1e3 * t_total / args.steps, "f64")
    sample = f"{per_step} of the {len(w.masses)} templates per step (evenly spread over the bank), full N={w.n} segment, p={w.p}"
    line["impl"] = "reference"
    line["config"]["units_per_step"] = per_step
    line["config"]["sample"] = sample
    line["cpu_baseline"] = {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    line["e2e"] = {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    line["gpu_launches"] = 0
    print(json.dumps(line), flush=True)
    return 0


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without a launcher: start N ranks (one per GPU) with torchrun and relay rank 0's line."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


STAGES = ("spectra", "pass1", "pass2", "chisq_at_events")
CHISQ_AT_TEXT = ("Eq. 5 evaluated from its definition at event samples: k_chisq_loud (every-sample mode: only events with "
                 "rho > 48 or in loud data, DESIGN.md reading 23) or k_chisq_at (chi^2 on demand: every event)")
STAGE_TEXT = {
    "decimated": {
        "spectra": "k_correlate_cm + k_bp_jobs + k_bandpower (5 kernels side by side) + k_uspec (template phasors x data, "
                   "coarse-grid band powers, U+); timed serialised, run beside the previous batch's passes on a side stream "
                   "in gwmf_filter",
        "pass1": "k_pass1_eff (first FFT pass of every effective band: writes n complex fp32 per n-point transform) "
                 "[+ k_prepass for bands of very many input rows: one more n complex written and read]",
        "pass2": "k_pass2_eff (last FFT stage + rho/chi^2/trigger epilogue: reads n complex fp32 per n-point transform)",
        "chisq_at_events": CHISQ_AT_TEXT},
    "two_pass": {
        "spectra": "-",
        "pass1": "k_pass1_narrow (pruned column FFT + first row stage, writes p*N*8 B/template) with the low-volume kernels "
                 "(k_correlate, k_pass1 generic, k_rowstage) beside it on the side stream; timed fork to join",
        "pass2": "k_pass2 (last FFT stage + rho/chi^2/trigger epilogue, reads p*N*8 B/template)",
        "chisq_at_events": CHISQ_AT_TEXT},
    "fused": {
        "spectra": "-",
        "pass1": "wide bands only: k_pass1 generic + k_rowstage (side stream; the next batch's correlates run beside k_fused)",
        "pass2": "k_fused (spill-free: narrow bands formed from the correlated spectrum, both row-transform stages, "
                 "rho/chi^2/trigger epilogue; no band intermediate in HBM)",
        "chisq_at_events": CHISQ_AT_TEXT},
}


def traffic_record(path, workload, stage):
    """ncu's dram__bytes_read.sum + dram__bytes_write.sum per template for a stage's kernel, from the committed
    capture summary profiles/traffic.json (written from the `ncu --set full` reports named inside it)."""
    fn = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(fn) as fh:
            rec = json.load(fh)
        ent = rec["entries"]["%s/%s/%s" % (workload, path, stage)]
        return float(ent["dram_bytes_per_template"]), "profiles/traffic.json: " + ent["source"]
    except Exception:
        return None, None


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_0906_4175_b200 import gwmf

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert world == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node {args.gpus}"
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    w, _ = load_workload(args.workload)
    seed_off, first, count = shard_plan(world, rank, len(w.masses), args.shard)
    w.seed += seed_off
    if w.config == 3:
        x = inputs.stream(w).astype(np.float32)
        segs = [np.ascontiguousarray(inputs.stream_segment(x, q, w.n)) for q in range(w.n_segments)]
    else:
        segs = [inputs.segment(w).astype(np.float32)]
    nseg = len(segs)
    s32 = segs[0]
    Sn = w.psd
    T = len(w.masses)

    f = gwmf.Filter(w.n, w.p, w.window, T, rho_thresh=w.rho_thresh, device=f"cuda:{local}", path=args.path, batch=args.batch,
                    chisq_on_demand=args.chisq_on_demand)
    path = f.path
    f.make_bank(w.masses)
    segs_dev = [torch.from_numpy(sg).to(dev) for sg in segs]
    sn_dev = torch.from_numpy(Sn).to(dev)
    if world > 1 and args.shard == "templates":
        for sd in segs_dev:                                  # one segment for everybody: rank 0's copy over NVLink
            dist.broadcast(sd, src=0)
    f.load_segment(segs_dev[0], sn_dev)

    def step_resident():
        out = None
        for q in range(nseg):
            if nseg > 1:
                f.load_segment(segs_dev[q])                  # device-resident segment, same PSD
            f.filter(first, count)
            out = f.triggers()
        return out

    try:
        uuid = str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid)
    for _ in range(max(args.warmup, 3) if nseg == 1 else max(min(args.warmup, 3), 1)):
        trig = step_resident()
    barrier()
    sampler.start()
    l0 = f.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(f.stream)
    for _ in range(args.steps):
        trig = step_resident()
    e1.record(f.stream)
    barrier()
    launches = f.launch_count - l0
    ms = reduce_max_ms(e0.elapsed_time(e1), dist if world > 1 else None, dev)
    value = world * count * nseg * args.steps / (ms * 1e-3) if args.shard == "segments" else T * nseg * args.steps / (ms * 1e-3)
    if world > 1 and args.shard == "templates":
        trig = gather_triggers(trig, dist, dev)              # the bank's event list of the last segment, on every rank
    f.load_segment(segs_dev[0])

    # per-stage device times (events inside the library, on its stream, stages serialised)
    reps = 3
    k_ms = np.zeros(4)
    k_launch = np.zeros(4)
    for _ in range(reps):
        m3, n3 = f.filter_timed(first, count)
        k_ms += m3
        k_launch += n3
    k_ms /= reps                                            # ms per step and stage
    k_launch /= reps
    transforms = f.transform_counts()[first:first + count]  # n-point transforms per template
    bytes_step = float(transforms.sum()) * w.n * 8.0        # pass 1 writes / pass 2 reads n complex fp32 per transform
    peak, peak_src = measured_peak()

    # end to end through the C ABI with HOST buffers: every segment is uploaded from pinned host memory inside the timed
    # region, overlapped with the filters of the segment before it (gwmf_load_segment with the PSD kept), and every
    # segment's events are read back:   filter(q); load(q + 1); triggers(q)
    segs_pin = [torch.from_numpy(sg).pin_memory() for sg in segs]
    f.load_segment(segs_pin[0], Sn)

    def step_e2e():
        out = None
        for q in range(nseg):
            f.filter(first, count)
            f.load_segment(segs_pin[(q + 1) % nseg])        # the next segment (of this or of the next step)
            out = f.triggers()
        return out

    for _ in range(3 if nseg == 1 else 1):
        trig_e = step_e2e()
    barrier()
    t0 = time.perf_counter()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(f.stream)
    d2h = 0
    for _ in range(args.steps):
        trig_e = step_e2e()
    g1.record(f.stream)
    barrier()
    wall_ms = (time.perf_counter() - t0) * 1e3
    ms_e2e = reduce_max_ms(max(g0.elapsed_time(g1), wall_ms), dist if world > 1 else None, dev)
    clocks = sampler.stop()
    units = world * count if args.shard == "segments" else T
    e2e_value = units * nseg * args.steps / (ms_e2e * 1e-3)
    f.load_segment(segs_dev[0])
    f.filter(first, count)
    f.synchronize()

    if rank == 0:
        line = base_line(args, w, value, ms / args.steps, "f32")
        line["config"]["path"] = path
        # SURVEY.md 8(f)-3 / PAPER.md:119,194 compares segment lengths in this unit: one template-segment is n / fs seconds
        line["template_seconds_of_data_per_s"] = value * w.n / w.fs
        if args.chisq_on_demand:
            line["metric"] += " -- chi^2 ON DEMAND (evaluated at the event samples only; not the headline workload)"
            line["config"]["chisq_mode"] = "on_demand"
        if nseg > 1:
            line["roofline_note"] = "per-stage times and bytes below are those of ONE segment (gwmf_filter_timed)"
        line["config"]["batch_templates_per_launch"] = float(count / max(k_launch[2], 1))
        line["config"]["n_point_transforms_per_template"] = float(transforms.mean())
        line["config"]["l2"] = ("no flush: every step streams the band intermediate (%.2f GB written by pass 1 and read by "
                                "pass 2 per step, %.0fx the 126 MB L2); the correlated spectra (%.0f MiB per launch) are "
                                "produced and consumed through L2 by design"
                                % (bytes_step / 1e9, bytes_step / 126e6, count / max(k_launch[2], 1) * w.n * 4 / 2**20))
        line["e2e"] = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(nseg * s32.nbytes),
                       "d2h_bytes_per_step": int(nseg * 12 + nseg * trig_e.nbytes), "ms_per_step": ms_e2e / args.steps,
                       "note": "per step: %d segment upload(s) from pinned host memory (the PSD is loaded once, before the timed "
                               "region, and kept), %d filter call(s), %d event read-back(s); uploads overlap the previous "
                               "segment's filters on the library's upload stream" % (nseg, nseg, nseg)}
        line["config"]["segments_per_step"] = nseg
        line["config"]["units_per_step"] = int(units * nseg)
        line["scaling"] = "weak" if args.shard == "segments" else "strong"
        line["config"]["shard"] = args.shard
        line["gpu_launches"] = int(launches)
        line["clocks"] = clocks
        if (clocks.get("samples") or 0) < 10:
            sys.stderr.write("bench.py: only %s clock samples in the timed regions: raise --steps for a record\n" % clocks.get("samples"))
        line["triggers_per_step"] = int(len(trig))
        kernels = {}
        for i, st in enumerate(STAGES):
            if k_launch[i] == 0:
                continue
            ent = {"kernel": STAGE_TEXT[path][st], "ms_per_step": float(k_ms[i]), "avg_launch_ms": float(k_ms[i] / k_launch[i]),
                   "share_of_step": float(k_ms[i] / k_ms.sum())}
            if st in ("pass1", "pass2") and path != "fused":
                ent["GB/s"] = bytes_step / (k_ms[i] * 1e-3) / 1e9
                ent["frac"] = ent["GB/s"] / peak
            kernels[st] = ent
        hbm_model = {"bytes_per_unit": 16.0 * w.p * w.n, "achieved": 16.0 * w.p * w.n * value / world / 1e9,
                     "frac": 16.0 * w.p * w.n * value / world / 1e9 / peak,
                     "note": "for comparison only: SURVEY.md 8(d3)'s two-pass model (16*p*N B per template-segment) at this "
                             "throughput; frac vs nominal 8 TB/s = %.3f.  The path that ran does not move these bytes"
                             % (16.0 * w.p * w.n * value / world / 8e12)}
        if path == "fused":
            # the spill-free kernel moves (almost) no HBM bytes: it is bound by the FP32 pipes and shared memory
            flops_unit = 5.0 * w.n * np.log2(w.n) * w.p            # p * 5 N log2 N per template-segment
            apeak, asrc = alu_peak()
            tfl = flops_unit * count / (k_ms[2] * 1e-3) / 1e12
            tr, tr_src = traffic_record(path, args.workload, "pass2")
            line["roofline"] = {
                "bound": "alu", "kernel": STAGE_TEXT[path]["pass2"], "achieved": float(tfl), "peak": apeak, "unit": "TFLOP/s",
                "frac": float(tfl / apeak), "peak_source": asrc,
                "peak_note": "a round-2 probe of packed fma.rn.f32x2 chains measured 68.1 TFLOP/s on this pool "
                             "(profiles/r2_fp32_peak.json); the probe is no longer part of the library",
                "flops": "dense-FFT equivalent (p*5N*log2N per unit), not executed flops",
                "traffic": tr * count / k_launch[2] if tr else None, "traffic_source": tr_src,
                "avg_launch_ms": float(k_ms[2] / k_launch[2]), "kernels": kernels, "hbm_model_equivalent": hbm_model}
        else:
            dom = "pass1" if k_ms[1] > k_ms[2] else "pass2"
            di = STAGES.index(dom)
            tr, tr_src = traffic_record(path, args.workload, dom)
            line["roofline"] = {
                "bound": "hbm", "kernel": STAGE_TEXT[path][dom], "achieved": kernels[dom]["GB/s"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dom]["frac"], "peak_source": peak_src,
                "bytes_per_launch": bytes_step / k_launch[di], "avg_launch_ms": float(k_ms[di] / k_launch[di]),
                "traffic": tr * count / k_launch[di] if tr else None, "traffic_source": tr_src,
                "kernels": kernels,
                "path": {"bytes_per_unit": 16.0 * w.n * float(transforms.mean()),
                         "achieved": 2 * bytes_step / ((k_ms[1] + k_ms[2]) * 1e-3) / 1e9,
                         "frac": 2 * bytes_step / ((k_ms[1] + k_ms[2]) * 1e-3) / 1e9 / peak,
                         "note": "both passes together: 16*N bytes per n-point transform that is run (%.2f per "
                                 "template-segment) over the summed device time of pass 1 and pass 2"
                                 % float(transforms.mean())},
                "hbm_model_equivalent": hbm_model}
        if not args.no_cpu_baseline and world == 1:
            cores = min(host_cores(), 32)
            nt = cores * (2 if cores <= 16 else 1)
            rate, dt = oracle_rate(w, s32.astype(np.float64), Sn, nt, cores)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{nt} of the {T} templates (evenly spread), full N={w.n} segment, "
                                              f"p={w.p}, {dt:.1f} s wall",
                                    "note": "the oracle as it stands: unoptimised fp64, own radix-2 FFT, p full-size "
                                            "transforms per template; a baseline, not a comparable CPU implementation",
                                    "context": "paper: 16x total speed-up, GeForce 8800 Ultra vs one 2.5 GHz Q9300 core "
                                               "(PAPER.md:5) -- other hardware, context only"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gwmf", choices=["gwmf", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="headline", choices=sorted(WORKLOADS))
    ap.add_argument("--path", default="auto", choices=["auto", "two_pass", "fused", "decimated"],
                    help="gwmf_params::path: auto = the library's choice (decimated for n >= 2^15)")
    ap.add_argument("--batch", type=int, default=0, help="templates per launch (0 = library default)")
    ap.add_argument("--chisq-on-demand", action="store_true",
                    help="gwmf_params::chisq_mode = ON_DEMAND: one full-band transform per template, chi^2 evaluated only at "
                         "the event samples (SURVEY.md 8(f)-2; a different workload from the headline's chi^2(t) at every sample)")
    ap.add_argument("--shard", default="segments", choices=["segments", "templates"],
                    help="N > 1: segments = every rank filters the whole bank against its own segment (weak scaling); "
                         "templates = one segment, the bank split by template id, events gathered (strong scaling)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
