#!/usr/bin/env python
"""bench.py — hydro cell-updates/s of the batched relaxing-TVD update on B200, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5|4|3]

One "step" = one pass of the whole hot path (H0-H9 of DESIGN.md: stage, three sweeps, store) over one batch:
one `gamer_hydro_advance` call on the workload.  Default workload = BASELINE.json configs[4] ("config 5": 32 768
patch groups, 134 M interior cells, 6.98 GB in / 2.68 GB out — the configuration the metric's roofline target is
quoted on), synthetic, filled on the device.  Inputs are far larger than L2 (126 MB), so every step streams from HBM.

Prints ONE JSON line (rank 0).  `value` = interior cell-updates per second, device-resident inputs, timed with
CUDA events on the launching stream; `e2e` = the same metric through `gamer_hydro_pipeline_run` with HOST (pinned)
buffers, host<->device copies inside the timed region.  N > 1 (torchrun): independent replicas, no collective on
the data path ("replicas only") — each rank advances its own copy of the workload.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_0907_3390_b200 import workloads as W  # noqa: E402

METRIC = "hydro cell-updates/sec (fp32) on 1 B200; % of roofline (HBM GB/s)"
UNIT = "cell-updates/s"
CELLS_PER_GROUP = 16 ** 3
BYTES_PER_GROUP = 212960 + 81920            # padded in + interior out
FLOPS_PER_GROUP = 1092 * 3474                # rows x flops per row, FMA = 2: the SMALLEST count
FP32_LANES_PER_SM = 128
PARITY_TOL = 1e-5                            # GPU vs fp32 oracle, metric R11 (north_star)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.sm_max = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
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
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        if not self.samples:
            return dict(sm_mhz=None, sm_max_mhz=self.sm_max, reasons=sorted(self.reasons), samples=0)
        return dict(sm_mhz=float(np.median(self.samples)), sm_max_mhz=self.sm_max, reasons=sorted(self.reasons),
                    samples=len(self.samples))


def kernel_source_hash(files=("rtvd_march.cuh", "hydro_kernel.cuh")):
    """sha256 (first 16 hex digits) over the CUDA sources of the fp32 hydro kernel (the row march and the kernel around
    it): identifies the kernel build that a profiles/*_traffic.csv row was captured on."""
    import hashlib
    h = hashlib.sha256()
    cdir = os.path.join(ROOT, "paper_0907_3390_b200", "csrc")
    for fn in files:
        h.update(fn.encode())
        h.update(open(os.path.join(cdir, fn), "rb").read())
    return h.hexdigest()[:16]


def profiled_traffic(config, n_groups, kernel="forward"):
    """(DRAM bytes per launch, source tag) of the hydro kernel from a committed ncu capture under profiles/ — only if the
    row names this workload AND was captured on the current kernel sources (kernel_src_sha16); else (None, why)."""
    import csv
    pdir = os.path.join(ROOT, "profiles")
    sha = kernel_source_hash()
    stale = None
    if os.path.isdir(pdir):
        for fn in sorted(os.listdir(pdir), reverse=True):
            if not fn.endswith("_traffic.csv"):
                continue
            with open(os.path.join(pdir, fn)) as f:
                for row in csv.DictReader(f):
                    if row.get("workload") != "config%d" % config or int(row["n_groups"]) != n_groups:
                        continue
                    if row.get("kernel", "forward") != kernel:
                        continue
                    if row.get("kernel_src_sha16") == sha:
                        return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]), \
                            "profiles/%s (ncu --set full, kernel sources %s)" % (fn, sha)
                    stale = "profiles/%s is of kernel sources %s, current %s" % (fn, row.get("kernel_src_sha16"), sha)
    return None, stale or "no ncu capture of this workload under profiles/"


def max_over_ranks(x, dist, device):
    """max of a python float over all ranks (identity without a process group); device = where the tensor lives."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(world, units_per_rank, seconds_max):
    """whole-job metric for independent replicas: all ranks' units over the slowest rank's time."""
    return world * units_per_rank / seconds_max


def physical_gpu_index(local):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


def make_device_workload(config, torch, device, n_override=None):
    """Returns (d_in, n_groups, dt, dh, gamma, description)."""
    if config == 5:
        n = n_override or W.CONFIG5["n_groups"]
        hot = W.config5_hot_groups(n)
        bg = torch.from_numpy(W.config5_group(False)).to(device)
        ht = torch.from_numpy(W.config5_group(True)).to(device)
        d_in = torch.empty((n, 5, 22, 22, 22), dtype=torch.float32, device=device)
        d_in[:] = bg
        d_in[torch.from_numpy(hot).to(device)] = ht
        return d_in, n, W.config5_dt(), W.CONFIG5["dh"], W.CONFIG5["gamma"], \
            "config5: %d groups, Sedov-like blast seeds in 1%% of groups (rho=1, p=1e-5, hot 2^3 cells p=1e3)" % n
    c = {4: W.config4, 3: W.config3}[config]()
    inp = c["inp"] if n_override is None else c["inp"][:n_override]
    d_in = torch.from_numpy(inp).to(device)
    return d_in, inp.shape[0], c["dt"], c["dh"], c["gamma"], "%s: %d groups" % (c["name"], inp.shape[0])


def time_advance(hydro, torch, stream, d_in, d_out, n, dt, dh, gamma, backward=0, steps=10, warmup=3):
    """mean ms per launch of one pass over n groups, CUDA events on `stream`."""
    for _ in range(warmup):
        hydro.gamer_hydro_advance_ex(d_in, d_out, n, 3, dt, dh, gamma, backward, stream=stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        hydro.gamer_hydro_advance_ex(d_in, d_out, n, 3, dt, dh, gamma, backward, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def cpu_sample(config, n_sample):
    """A bounded sample of the same workload for the oracle: the first n_sample groups (config 5 keeps its 1 % hot)."""
    if config == 5:
        c = W.config5(range(n_sample))
    else:
        c = {4: W.config4, 3: W.config3}[config]()
        c["inp"] = c["inp"][:n_sample]
    return c


def time_oracle(config, cores, target_core_seconds=20.0, n_sample=None):
    import oracle
    probe = cpu_sample(config, 32)
    t0 = time.perf_counter()
    oracle.hydro_advance(probe["inp"], probe["dt"], probe["dh"], probe["gamma"], n_threads=1, return_bad=True)
    per_group = (time.perf_counter() - t0) / 32
    if n_sample is None:
        n_sample = int(max(8, min(8192, target_core_seconds / per_group)))
    c = cpu_sample(config, n_sample)
    n_sample = c["inp"].shape[0]
    t0 = time.perf_counter()
    c["out"] = oracle.hydro_advance(c["inp"], c["dt"], c["dh"], c["gamma"], n_threads=cores, return_bad=True)[0]
    wall = time.perf_counter() - t0
    return dict(value=n_sample * CELLS_PER_GROUP / wall, unit=UNIT, cores=cores, kind="oracle",
                sample="first %d groups of the workload, fp32 oracle, %d OpenMP threads over groups, %.2f s wall"
                       % (n_sample, cores, wall)), c, wall


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    import oracle
    # each step is a bounded sample sized so that the whole --steps/--warmup run ends within about two minutes
    per_step_wall = min(1.5, 120.0 / max(1, args.steps + args.warmup))
    _, c, _ = time_oracle(args.config, cores, target_core_seconds=per_step_wall * cores)
    n_sample = c["inp"].shape[0]
    for _ in range(args.warmup):
        oracle.hydro_advance(c["inp"], c["dt"], c["dh"], c["gamma"], n_threads=cores, return_bad=True)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.hydro_advance(c["inp"], c["dt"], c["dh"], c["gamma"], n_threads=cores, return_bad=True)
    wall = time.perf_counter() - t0
    value = args.steps * n_sample * CELLS_PER_GROUP / wall
    sample = "each step = first %d groups of the workload (bounded sample), fp32 oracle, %d OpenMP threads" % (n_sample, cores)
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * wall / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f32", data="synthetic", impl="reference",
                config=dict(workload="config%d" % args.config, sample_groups=n_sample),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    from paper_0907_3390_b200 import hydro, probes

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)

    hydro.lib()     # fail loudly here if the CUDA library is missing
    peaks = load_peaks()
    d_in, n, dt, dh, gamma, desc = make_device_workload(args.config, torch, device, args.groups)
    d_out = torch.empty((n, 5, 16, 16, 16), dtype=torch.float32, device=device)
    info = hydro.gamer_hydro_launch_info(n)
    stream = torch.cuda.current_stream()

    def step():
        hydro.gamer_hydro_advance(d_in, d_out, n, 3, dt, dh, gamma, stream=stream)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    evs[0].record(stream)
    for i in range(args.steps):
        step()
        evs[i + 1].record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    if dist is not None:
        dist.barrier()
    total_ms = evs[0].elapsed_time(evs[-1])
    per_launch_ms = [evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)]
    total_ms = max_over_ranks(total_ms, dist, device)
    ms_per_step = total_ms / args.steps
    value = job_throughput(world, n * CELLS_PER_GROUP, ms_per_step * 1e-3)
    kernel_ms = float(np.mean(per_launch_ms))

    # CPU baseline leg: the oracle as it stands on the host cores, on the first groups of the same workload.  Its
    # output doubles as a check of the timed output on those groups: a wrong-but-fast run makes bench.py exit 1.
    cpu_baseline, parity, cpu_1thread, failed = None, None, None, []
    if rank == 0 and world == 1 and not args.no_cpu:
        cores = os.cpu_count() or 1
        cpu_baseline, cs, _ = time_oracle(args.config, cores)
        if not args.no_check:
            ns = cs["out"].shape[0]
            parity = W.parity_error(d_out[:ns].cpu().numpy(), cs["out"], gamma)["max_rel"]
            cpu_baseline["parity_max_rel_on_sample"] = parity
            if not parity <= PARITY_TOL:
                failed.append("parity on the first %d groups: %.3g > %.0e" % (ns, parity, PARITY_TOL))
        # the plain oracle, fp32, ONE thread, on config 3 (512 groups)
        import oracle
        c3 = W.config3()
        t0 = time.perf_counter()
        oracle.hydro_advance(c3["inp"], c3["dt"], c3["dh"], c3["gamma"], n_threads=1)
        w3 = time.perf_counter() - t0
        cpu_1thread = dict(value=c3["inp"].shape[0] * CELLS_PER_GROUP / w3, unit=UNIT, cores=1, kind="oracle",
                           sample="config3, all %d groups, fp32 oracle, 1 thread, %.2f s wall" % (c3["inp"].shape[0], w3))
        del c3

    # roofline of the one kernel of the step
    n_sm = torch.cuda.get_device_properties(device).multi_processor_count
    fp32_peak_tflops = n_sm * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    ach_gbs = n * BYTES_PER_GROUP / (kernel_ms * 1e-3) / 1e9
    ach_tf = n * FLOPS_PER_GROUP / (kernel_ms * 1e-3) / 1e12
    roofline_hbm = dict(bound="hbm", achieved=ach_gbs, peak=peaks["hbm_gbs"], unit="GB/s", frac=ach_gbs / peaks["hbm_gbs"],
                        traffic=None, peak_source=peaks["source"])
    roofline_alu = dict(bound="alu", achieved=ach_tf, peak=fp32_peak_tflops, unit="TFLOP/s", frac=ach_tf / fp32_peak_tflops,
                        traffic=None, peak_source="derived: %d SM x 128 FP32 lanes x 2 x sm_max_mhz (DESIGN.md); `frac` "
                                                  "uses this one, the measured FMA rate is beside it" % n_sm)
    # the FMA-only micro-benchmark of the library, measured in this run
    d_sink = torch.zeros(4, dtype=torch.float32, device=device)
    peak_meas_tf, peak_meas_lanes = probes.gamer_probe_fp32_peak(5, d_sink, peaks["sm_max_mhz"])
    roofline_alu["peak_measured_tflops"] = peak_meas_tf
    roofline_alu["peak_measured_fma_per_clk_per_sm"] = peak_meas_lanes
    roofline_alu["frac_of_measured_peak"] = ach_tf / peak_meas_tf
    # what the instruction mix of the march costs in steady state: clocks per warp-march and sub-partition
    # slot with 1..4 warps per sub-partition, no loads, no barriers; and the cost of an FMA with three distinct registers
    issue_probe = None
    if rank == 0:
        ffma3 = probes.gamer_probe_issue(0, 4)
        march = {ax: [probes.gamer_probe_issue(i + 1, k) for k in (1, 2, 3, 4)] for i, ax in enumerate("xyz")}
        # a group is 16 x-, 11 y-, 8 z-marches on 4 sub-partitions: with every slot filled at the 4-warp rate
        packed = (16 * march["x"][3] + 11 * march["y"][3] + 8 * march["z"][3]) / 4.0
        # the kernel's three phases run 4, 3 and 2 warps per sub-partition
        phases = 4 * march["x"][3] + 3 * march["y"][2] + 2 * march["z"][1]
        clk = peaks["sm_max_mhz"] * 1e6
        issue_probe = dict(api="gamer_probe_issue (libgamer_probes.so)", ffma_3_distinct_registers_clocks_per_instr=ffma3,
                           clocks_per_warp_march_by_warps_per_subpartition=march,
                           ns_per_group_if_every_slot_ran_at_the_4_warp_rate=packed / clk * 1e9 / n_sm,
                           ns_per_group_sum_of_the_three_phases=phases / clk * 1e9 / n_sm)
    # the metric's roofline is the slower of the two bounds (north_star): FP32 at 51 ns/group vs HBM at 45 ns/group
    t_alu = FLOPS_PER_GROUP / (fp32_peak_tflops * 1e12)
    t_hbm = BYTES_PER_GROUP / (peaks["hbm_gbs"] * 1e9)
    roofline = dict(roofline_alu if t_alu >= t_hbm else roofline_hbm)
    traffic, traffic_source = profiled_traffic(args.config, n)
    for r in (roofline, roofline_hbm, roofline_alu):
        r["traffic"] = traffic
        r["traffic_source"] = traffic_source
    roofline["algorithmic_bytes"] = n * BYTES_PER_GROUP
    roofline["algorithmic_flops"] = n * FLOPS_PER_GROUP
    roofline["flops_per_group"] = FLOPS_PER_GROUP
    roofline["flops_count"] = ("hand count 1092 rows x 3474 (SURVEY 8(d)), the smallest of three: the kernel's own "
                               "formulation is 3492 per row, the oracle's literal Eq.8 counts 5.33 M per group")
    roofline["kernel_ms"] = kernel_ms
    roofline["ns_per_group"] = kernel_ms * 1e6 / n

    # fp32 backward pass (z,y,x), same workload: half of every forward+backward step of the paper (:174-176)
    backward = None
    if rank == 0:
        ms_b = time_advance(hydro, torch, stream, d_in, d_out, n, dt, dh, gamma, backward=1, steps=10)
        backward = dict(ns_per_group=ms_b * 1e6 / n, ratio_to_forward=ms_b / kernel_ms,
                        frac=(n * FLOPS_PER_GROUP / (ms_b * 1e-3) / 1e12) / fp32_peak_tflops)
        hydro.gamer_hydro_advance(d_in, d_out, n, 3, dt, dh, gamma, stream=stream)      # d_out = the forward result again
        torch.cuda.synchronize()

    # config 4 (the arithmetic-realistic input): as specified (4096 groups) and tiled to 32 768 groups
    config4 = None
    if rank == 0 and world == 1 and args.config == 5 and not args.no_config4:
        c4 = W.config4()
        n4 = c4["inp"].shape[0]
        d4 = torch.from_numpy(c4["inp"]).to(device)
        o4 = torch.empty((n4, 5, 16, 16, 16), dtype=torch.float32, device=device)
        ms4 = time_advance(hydro, torch, stream, d4, o4, n4, c4["dt"], c4["dh"], c4["gamma"], steps=20)
        config4 = dict(workload="config4: %d groups (lognormal density, sigma(ln rho) = 2, reading R17)" % n4,
                       n_groups=n4, ns_per_group=ms4 * 1e6 / n4,
                       frac=(n4 * FLOPS_PER_GROUP / (ms4 * 1e-3) / 1e12) / fp32_peak_tflops)
        if not args.no_cpu and not args.no_check:
            import oracle
            ns4 = 512
            ref4 = oracle.hydro_advance(c4["inp"][:ns4], c4["dt"], c4["dh"], c4["gamma"], n_threads=os.cpu_count() or 1)
            p4 = W.parity_error(o4[:ns4].cpu().numpy(), ref4, c4["gamma"])["max_rel"]
            config4["parity_max_rel_on_first_%d_groups" % ns4] = p4
            if not p4 <= PARITY_TOL:
                failed.append("config 4 parity: %.3g > %.0e" % (p4, PARITY_TOL))
        rep = n // n4
        if rep > 1 and n4 * rep * (BYTES_PER_GROUP) < 12e9:
            d4r = d4.repeat(rep, 1, 1, 1, 1)
            o4r = torch.empty((n4 * rep, 5, 16, 16, 16), dtype=torch.float32, device=device)
            sampler4 = ClockSampler(physical_gpu_index(local), period=0.005)
            sampler4.start()
            ms4r = time_advance(hydro, torch, stream, d4r, o4r, n4 * rep, c4["dt"], c4["dh"], c4["gamma"], steps=40)
            clocks4 = sampler4.stop()
            config4["tiled_x%d" % rep] = dict(n_groups=n4 * rep, ns_per_group=ms4r * 1e6 / (n4 * rep),
                                              frac=(n4 * rep * FLOPS_PER_GROUP / (ms4r * 1e-3) / 1e12) / fp32_peak_tflops,
                                              ratio_to_config5=(ms4r / (n4 * rep)) / (kernel_ms / n), clocks=clocks4)
            del d4r, o4r
        del d4, o4, c4
        torch.cuda.empty_cache()

    # end to end through the public C-ABI call with host buffers
    e2e = None
    if (rank == 0 or world > 1) and not args.no_e2e:
        try:
            h_in = torch.empty(d_in.shape, dtype=torch.float32, pin_memory=True)
            h_out = torch.empty(d_out.shape, dtype=torch.float32, pin_memory=True)
            h_in.copy_(d_in)
            torch.cuda.synchronize()
            e2e_steps = max(1, min(args.steps, args.e2e_steps))
            chunk, ns = args.chunk, args.streams
            hydro.gamer_hydro_pipeline_run(h_in, h_out, n, 3, dt, dh, gamma, 0, chunk, ns)      # warm-up
            if dist is not None:
                dist.barrier()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                hydro.gamer_hydro_pipeline_run(h_in, h_out, n, 3, dt, dh, gamma, 0, chunk, ns)
            wall = time.perf_counter() - t0
            wall = max_over_ranks(wall, dist, device)
            e2e = dict(value=job_throughput(world, e2e_steps * n * CELLS_PER_GROUP, wall), unit=UNIT,
                       h2d_bytes_per_step=int(h_in.numel() * 4), d2h_bytes_per_step=int(h_out.numel() * 4),
                       steps=e2e_steps, ms_per_step=1e3 * wall / e2e_steps, groups_per_chunk=chunk, n_streams=ns,
                       h2d_gbs=h_in.numel() * 4 * e2e_steps / wall / 1e9, api="gamer_hydro_pipeline_run (pinned host)")
            e2e["d2h_gbs"] = h_out.numel() * 4 * e2e_steps / wall / 1e9
            # The pipeline's own report (SURVEY.md 8(d) "Pipeline subsystem"; PAPER.md:354-356 Fig.5, :368): the link
            # measured in the same run on the same pinned buffers, then one pass per (N_g, N_s) point.
            if world == 1 and not args.no_pipeline_sweep:
                def copy_ms(pairs):
                    """[(dst, src, stream)] started together; returns ms until the last one is done (device events)."""
                    torch.cuda.synchronize()
                    ev = []
                    for dst, src, st in pairs:
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        with torch.cuda.stream(st):
                            e0.record(st)
                            dst.copy_(src, non_blocking=True)
                            e1.record(st)
                        ev.append((e0, e1))
                    torch.cuda.synchronize()
                    return max(ev[0][0].elapsed_time(e1) for _, e1 in ev)
                s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
                in_b, out_b = h_in.numel() * 4, h_out.numel() * 4
                copy_ms([(d_in, h_in, s1)])                                            # warm-up (h_in holds d_in's data)
                t_h2d = min(copy_ms([(d_in, h_in, s1)]) for _ in range(2))
                t_d2h = min(copy_ms([(h_out, d_out, s2)]) for _ in range(2))
                t_both = min(copy_ms([(d_in, h_in, s1), (h_out, d_out, s2)]) for _ in range(2))
                link = dict(h2d_alone_gbs=in_b / t_h2d / 1e6, d2h_alone_gbs=out_b / t_d2h / 1e6,
                            both_at_once_ms=t_both, both_at_once_h2d_gbs=in_b / t_both / 1e6,
                            both_at_once_d2h_gbs=out_b / t_both / 1e6, api="pinned cudaMemcpyAsync (torch copy_)")
                points = [(chunk, 1), (chunk, 2), (chunk, 4), (1024, 4), (2048, 4), (4096, 4)]
                sweep = []
                for ng, nst in points:
                    ng = min(ng, n)
                    hydro.gamer_hydro_pipeline_run(h_in, h_out, n, 3, dt, dh, gamma, 0, ng, nst)      # staging grows here
                    t0 = time.perf_counter()
                    hydro.gamer_hydro_pipeline_run(h_in, h_out, n, 3, dt, dh, gamma, 0, ng, nst)
                    w = (time.perf_counter() - t0) * 1e3
                    # what a perfect overlap leaves: the longest of the three serial sums (copies at the alone rates)
                    sweep.append(dict(groups_per_chunk=ng, n_streams=nst, wall_ms=w, h2d_gbs=in_b / w / 1e6,
                                      d2h_gbs=out_b / w / 1e6, sum_h2d_ms=t_h2d, sum_kernel_ms=kernel_ms, sum_d2h_ms=t_d2h,
                                      overlap_efficiency=max(t_h2d, kernel_ms, t_d2h) / w,
                                      serial_ms=t_h2d + kernel_ms + t_d2h))
                e2e["pipeline"] = dict(link=link, sweep=sweep,
                                       note="overlap_efficiency = max(sum H2D, sum kernel, sum D2H) / wall; the sums are "
                                            "the whole batch at the alone-measured rates and the device-timed kernel")
            del h_in, h_out
            hydro.gamer_hydro_pipeline_release()
        except Exception as ex:      # e.g. not enough pinnable host memory
            e2e = dict(value=None, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0, error=str(ex)[:200])

    # NEXT-1/2 (reported separately): the same forward pass with the optional outputs switched on
    optional_outputs = None
    if rank == 0 and not args.no_ghost_fill:
        d_face = torch.empty((n, 3, 3, 5, 16, 16), dtype=torch.float32, device=device)
        d_speed = torch.empty((n,), dtype=torch.float32, device=device)
        optional_outputs = {}
        for name, kw in (("maxspeed", dict(d_group_maxspeed=d_speed)),
                         ("face_flux+maxspeed", dict(d_face_flux=d_face, d_group_maxspeed=d_speed))):
            for _ in range(2):
                hydro.gamer_hydro_advance_ex(d_in, d_out, n, 3, dt, dh, gamma, 0, stream=stream, **kw)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(5):
                hydro.gamer_hydro_advance_ex(d_in, d_out, n, 3, dt, dh, gamma, 0, stream=stream, **kw)
            e1.record(stream)
            torch.cuda.synchronize()
            optional_outputs[name] = dict(ns_per_group=e0.elapsed_time(e1) / 5 * 1e6 / n)
        del d_face, d_speed

    # NEXT-4 (reported separately): the forward pass in double precision on the first 8192 groups of the workload
    f64 = None
    if rank == 0 and not args.no_ghost_fill:
        n64 = min(n, 8192)
        d_in64 = d_in[:n64].double()
        d_out64 = torch.empty((n64, 5, 16, 16, 16), dtype=torch.float64, device=device)
        for _ in range(2):
            hydro.gamer_hydro_advance_f64_ex(d_in64, d_out64, n64, 3, dt, dh, gamma, stream=stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(5):
            hydro.gamer_hydro_advance_f64_ex(d_in64, d_out64, n64, 3, dt, dh, gamma, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms64 = e0.elapsed_time(e1) / 5
        gbs64 = n64 * 2 * BYTES_PER_GROUP / (ms64 * 1e-3) / 1e9
        e0.record(stream)
        for _ in range(3):
            hydro.gamer_hydro_advance_f64_ex(d_in64, d_out64, n64, 3, dt, dh, gamma, backward=1, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms64b = e0.elapsed_time(e1) / 3
        # the same pass with face fluxes and per-group CFL speed in double (gamer_hydro_advance_f64_ex)
        d_face64 = torch.empty((n64, 3, 3, 5, 16, 16), dtype=torch.float64, device=device)
        d_spd64 = torch.empty((n64,), dtype=torch.float64, device=device)
        for _ in range(2):
            hydro.gamer_hydro_advance_f64_ex(d_in64, d_out64, n64, 3, dt, dh, gamma, 0, d_face64, d_spd64, stream=stream)
        eo0, eo1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        eo0.record(stream)
        for _ in range(3):
            hydro.gamer_hydro_advance_f64_ex(d_in64, d_out64, n64, 3, dt, dh, gamma, 0, d_face64, d_spd64, stream=stream)
        eo1.record(stream)
        torch.cuda.synchronize()
        ms64_opt = eo0.elapsed_time(eo1) / 3
        del d_face64, d_spd64
        f64 = dict(api="gamer_hydro_advance_f64_ex", n_groups=n64, ns_per_group=ms64 * 1e6 / n64,
                   ns_per_group_with_face_flux_and_maxspeed=ms64_opt * 1e6 / n64,
                   backward_ns_per_group=ms64b * 1e6 / n64,
                   value=n64 * CELLS_PER_GROUP / (ms64 * 1e-3), unit=UNIT, dtype="f64",
                   hbm_achieved_gbs=gbs64, hbm_frac=gbs64 / peaks["hbm_gbs"], algorithmic_bytes=n64 * 2 * BYTES_PER_GROUP)
        del d_in64, d_out64

    # NEXT-3 (reported separately, not part of the step): device-side ghost fill of the same batch seen as a periodic
    # box of groups — reads every interior once, writes every padded group once.  It overwrites d_in, so it runs last.
    ghost_fill = None
    if rank == 0 and not args.no_ghost_fill:
        gxyz = round(n ** (1.0 / 3.0))
        box = (gxyz, gxyz, gxyz) if gxyz ** 3 == n else (n, 1, 1)
        for _ in range(2):
            hydro.gamer_hydro_ghost_fill(d_out, d_in, box[0], box[1], box[2], stream=stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(5):
            hydro.gamer_hydro_ghost_fill(d_out, d_in, box[0], box[1], box[2], stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        gf_ms = e0.elapsed_time(e1) / 5
        gf_gbs = n * BYTES_PER_GROUP / (gf_ms * 1e-3) / 1e9
        ghost_fill = dict(api="gamer_hydro_ghost_fill", box_groups=list(box), ms=gf_ms, bound="hbm", achieved=gf_gbs,
                          peak=peaks["hbm_gbs"], unit="GB/s", frac=gf_gbs / peaks["hbm_gbs"],
                          algorithmic_bytes=n * BYTES_PER_GROUP)

        # a thin box: 1024 groups as 256 x 4 x 1 give 20 strips, far fewer than SMs; the walk along x
        # is cut into segments so that the launch still fills the GPU
        if n >= 1024:
            tb = (256, 4, 1)
            for _ in range(2):
                hydro.gamer_hydro_ghost_fill(d_out, d_in, tb[0], tb[1], tb[2], stream=stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(5):
                hydro.gamer_hydro_ghost_fill(d_out, d_in, tb[0], tb[1], tb[2], stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            tb_ms = e0.elapsed_time(e1) / 5
            ghost_fill["thin_box"] = dict(box_groups=list(tb), ms=tb_ms, achieved=1024 * BYTES_PER_GROUP / (tb_ms * 1e-3) / 1e9,
                                          unit="GB/s", note="302 MB: partly L2-resident, compare with itself across rounds")
            hydro.gamer_hydro_ghost_fill(d_out, d_in, box[0], box[1], box[2], stream=stream)   # restore the full box

    # NEXT-3 driver: whole steps (dt, forward pass, ghost fill) without leaving the device; runs last, it evolves d_in
    run_uniform = None
    if ghost_fill is not None:
        box = ghost_fill["box_groups"]
        d_work = torch.zeros(4 + n, dtype=torch.float32, device=device)
        d_log = torch.zeros(16, dtype=torch.float32, device=device)

        def timed_steps(fn, second, k):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn(d_in, second, box[0], box[1], box[2], 0, 0, 0, k, 0, 0.5, dh, gamma, d_work, d_log, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1)

        # a call = one pass of Eq.30 over the initial state + k steps: the per-step time is the difference of two calls
        timed_steps(hydro.gamer_hydro_run_uniform, d_out, 1)
        t2, t6 = timed_steps(hydro.gamer_hydro_run_uniform, d_out, 2), timed_steps(hydro.gamer_hydro_run_uniform, d_out, 6)
        ru_ms = (t6 - t2) / 4
        run_uniform = dict(api="gamer_hydro_run_uniform", steps="(6-step call - 2-step call) / 4", ms_per_step=ru_ms,
                           ms_first_call_overhead=t2 - 2 * ru_ms,
                           value=n * CELLS_PER_GROUP / (ru_ms * 1e-3), unit=UNIT,
                           dt_finite=bool(torch.isfinite(d_log).all().item()))

    if rank == 0:
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                    ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                    data="synthetic",
                    config=dict(workload=desc, n_groups=n, cells_per_group=CELLS_PER_GROUP, parallelism="replicas x%d" % world,
                                l2="inputs (%.2f GB) larger than L2; no flush needed" % (d_in.numel() * 4 / 1e9),
                                launch=info),
                    roofline=roofline, roofline_hbm=roofline_hbm, roofline_alu=roofline_alu,
                    cpu_baseline=cpu_baseline, cpu_baseline_1thread=cpu_1thread, e2e=e2e, gpu_launches=args.steps,
                    clocks=clocks, backward=backward, issue_probe=issue_probe, config4=config4, failed=failed,
                    next3_ghost_fill=ghost_fill, next12_optional_outputs=optional_outputs, next4_f64=f64, next3_run_uniform=run_uniform,
                    parity_spot_check_max_rel=parity)
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    if failed:
        print("bench.py: FAILED: " + "; ".join(failed), file=sys.stderr)
        return 1
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=[3, 4, 5])
    ap.add_argument("--groups", type=int, default=None, help="debug: override the number of groups")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--chunk", type=int, default=512, help="pipeline: groups per chunk (N_g)")
    ap.add_argument("--streams", type=int, default=3, help="pipeline: number of streams (N_s)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer pipeline leg (profiling runs)")
    ap.add_argument("--no-pipeline-sweep", action="store_true",
                    help="skip the pipeline's own report (link rates, N_g x N_s sweep) inside the e2e leg")
    ap.add_argument("--no-check", action="store_true")
    ap.add_argument("--no-config4", action="store_true", help="skip the config-4 sub-record")
    ap.add_argument("--no-ghost-fill", action="store_true", help="skip the separate ghost-fill measurement")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
