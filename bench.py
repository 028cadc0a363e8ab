#!/usr/bin/env python
"""bench.py -- walker-steps/s of the whole RMS hot path on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Workload (config.workload): the cfg4 throughput point of BASELINE.json on the synthetic mouse-like axon
substrate of cfg2 -- 500x500x2000 uint16 lattice, ~300 axons, 1e6 intra-axonal walkers x 10,000 Monte Carlo
steps, PGSE with 60 directions x 11 b-values, impermeable membranes, D = 2 um^2/ms, dt = 2e-4 ms.
One bench "step" is one pass of the whole path: rms_substrate_create (neighbourhood lattice built from labels
resident in HBM) -> rms_walkers_init -> rms_run (walk, phase/T2 accumulation, moment and signal reductions,
normalisation).  `value` = walker-steps/s with the labels already in HBM; `e2e` = the same through the C ABI
from pinned HOST labels (host->device copy and result read-back inside the timed region).

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

# Algorithmic thread-instructions per walker-step, frozen in DESIGN.md ("Roofline") before tuning.
ALGORITHMIC_INSTR_PER_STEP = 80.0
N_SM, LANES_PER_SM = 148, 128          # B200: 4 schedulers x 32 lanes per SM, one warp instruction per clock each
# DRAM traffic of the step kernel per launch (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture),
# by the configuration that was captured; a run of any other configuration reports traffic = null.
# key: (substrate, lattice, layout, lattice_format, walkers, mc_steps, fp64)
NCU_CAPTURES = {
    # RMS_LAYOUT_AUTO picks z fastest on this lattice: the two keys name the same launch
    ("cfg4", "facemask", "auto", "oct", 1_000_000, 10_000, False): {"bytes": 40.94e9, "source": "profiles/r2j_step_fast_ncu.md (40.04 GB read + 0.91 GB written)"},
    ("cfg4", "facemask", "z", "oct", 1_000_000, 10_000, False): {"bytes": 40.94e9, "source": "profiles/r2j_step_fast_ncu.md (40.04 GB read + 0.91 GB written)"},
    ("cfg4", "facemask", "auto", "dict", 1_000_000, 10_000, False): {"bytes": 6.93e9, "source": "profiles/r2k_step_fast_dict_ncu.md (6.09 GB read + 0.84 GB written)"},
    ("cfg4", "facemask", "z", "dict", 1_000_000, 10_000, False): {"bytes": 6.93e9, "source": "profiles/r2k_step_fast_dict_ncu.md (6.09 GB read + 0.84 GB written)"},
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--walkers", type=int, default=1_000_000)
    ap.add_argument("--mc-steps", type=int, default=10_000)
    ap.add_argument("--dirs", type=int, default=60)
    ap.add_argument("--lattice", default="facemask", choices=["facemask", "labels"])
    ap.add_argument("--scale", default="full", choices=["full", "test"])
    ap.add_argument("--layout", default="auto", choices=["auto", "x", "z"],
                    help="memory order of the neighbourhood lattice (auto: RMS_LAYOUT_AUTO picks the axis the membranes run along)")
    ap.add_argument("--lattice-format", default="dict", choices=["oct", "dict"],
                    help="dict: RMS_LATTICE_DICT, 2-byte code per voxel + dictionary of octant words (the faster step kernel on "
                         "this workload, a quarter of the memory and a sixth of the DRAM traffic); oct: 8-byte octant word per "
                         "voxel, the C ABI's default (a build 1.2 ms shorter)")
    ap.add_argument("--waves", type=int, default=1,
                    help="number of PGSE waveforms evaluated on the same trajectories (sequence sweep, not the headline)")
    ap.add_argument("--substrate", default="cfg4", choices=["cfg4", "cfg3"],
                    help="cfg3: the permeable, D- and T2-contrast variant of the lattice with walkers in every label (not the headline)")
    ap.add_argument("--fp64", action="store_true", help="RMS_RUN_FP64: the step kernel in fp64 arithmetic (not the headline)")
    ap.add_argument("--interaction", default="ec", choices=["ec", "rs", "erl"],
                    help="membrane interaction: elastic collision (the method, the headline), rejection sampling, equal-step-length random leap")
    ap.add_argument("--general-kernel", action="store_true", help="RMS_RUN_GENERAL_KERNEL (diagnostic)")
    ap.add_argument("--no-slices", action="store_true", help="RMS_RUN_NO_SLICES: one block per group of walkers for the whole launch (diagnostic)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-walkers", type=int, default=250_000)
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json configs[4]: walkers 1e5..1e8 x {1, 60} directions x {neighbourhood lattice, label "
                         "gather}, one JSON line per point (not part of the driver contract)")
    ap.add_argument("--sweep-max-walkers", type=int, default=100_000_000)
    return ap.parse_args()


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md recipe).  Sampled in-process through
    NVML (nvidia_ml_py) every 50 ms; an external `nvidia-smi -lms` loop contends for the driver lock with the
    path's own calls and was measured to slow a pass by tens of ms.  Falls back to nvidia-smi if NVML is missing."""
    NAMES = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines, self.samples = index, None, [], []
        self.stop_flag = threading.Event()
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(self._physical_index(index))
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nvml = None

    @staticmethod
    def _physical_index(index):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            ids = [v.strip() for v in vis.split(",") if v.strip()]
            if index < len(ids) and ids[index].isdigit():
                return int(ids[index])
        return index

    def start(self):
        if self.nvml:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "250",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _poll(self):
        n = self.nvml
        while not self.stop_flag.is_set():
            try:
                sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                pw = n.nvmlDeviceGetPowerUsage(self.handle) / 1000.0
                try:
                    rs = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
                except Exception:
                    rs = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                self.samples.append((sm, pw, rs))
            except Exception:
                pass
            self.stop_flag.wait(0.05)

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.nvml:
            self.stop_flag.set()
            self.thread.join(timeout=2)
            sm = [x[0] for x in self.samples]
            reasons = sorted(nm for nm, bit in self.NAMES.items() if any(x[2] & bit for x in self.samples))
            return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": self.sm_max,
                    "power_w_max": max((x[1] for x in self.samples), default=None), "samples": len(sm), "reasons": reasons,
                    "source": "nvml, 50 ms"}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons),
                "source": "nvidia-smi -lms 250"}


def make_workload(args):
    import rms_inputs as ri
    cfg = ri.make_config("cfg4", args.scale, n_walkers=args.walkers, n_steps=args.mc_steps, n_dir=args.dirs)
    if args.substrate == "cfg3":
        cfg.substrate = ri.make_config("cfg3", args.scale).substrate
    if args.waves > 1:      # sequence sweep: waveform m has delta = Delta / (m + 1) ... all on one set of trajectories
        seq = cfg.sequence
        n = seq.n_steps
        waves = np.stack([ri.pgse_wave(n, max(1, int(0.4 * n / (m + 1))), int(0.6 * n)) for m in range(args.waves)])
        gamp = np.repeat(seq.gamp, args.waves, axis=0)
        cfg.sequence = dataclasses.replace(seq, wave=waves.astype(np.float32), gamp=gamp)
    return cfg


def workload_config(args, cfg, extra=None):
    nx, ny, nz = cfg.substrate.shape_xyz
    c = {"workload": "cfg4 point on the cfg2 synthetic axon substrate (BASELINE.json configs[4] on configs[2])",
         "lattice": f"{nx}x{ny}x{nz} uint16", "n_axons": cfg.substrate.meta.get("n_axons"),
         "intra_fraction": round(cfg.substrate.meta.get("intra_fraction", 0.0), 4),
         "walkers_per_gpu": args.walkers, "mc_steps": args.mc_steps, "dt_ms": cfg.sequence.dt_ms,
         "directions": int(cfg.sequence.dirs.shape[0]), "b_values": int(cfg.sequence.gamp.shape[1]),
         "lattice_path": args.lattice, "layout": args.layout, "lattice_format": args.lattice_format,
         "interaction": args.interaction, "pass": "rms_substrate_create + rms_walkers_init + rms_run",
         "l2": ("inputs larger than L2 (label lattice 1.0 GB + " + ("code lattice 1.0 GB" if args.lattice_format == "dict" else "octant lattice 4.0 GB") +
                " vs 126 MB L2)") if args.scale == "full"
         else "reduced test lattice (fits L2) -- not a valid bench configuration"}
    if extra:
        c.update(extra)
    return c


def run_reference(args):
    """The CPU oracle as it stands, on the host cores, on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = make_workload(args)
    threads = oracle.rms_oracle.default_threads()
    sample = min(args.cpu_sample_walkers, args.walkers)
    oracle.build()
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.run(cfg.substrate, cfg.sequence, sample, cfg.seed, first_id=0, n_threads=threads)
        t1 = time.perf_counter()
        if it >= args.warmup:
            times.append(t1 - t0)
    total = sum(times)
    value = sample * args.mc_steps * len(times) / total
    line = {"impl": "reference", "metric": "walker_steps_per_s", "value": value, "unit": "walker-steps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, cfg),
            "cpu_baseline": {"value": value, "unit": "walker-steps/s", "cores": threads, "kind": "oracle",
                             "sample": f"first {sample} walker ids x {args.mc_steps} steps"},
            "e2e": {"value": value, "unit": "walker-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_sweep(args):
    """Throughput sweep of BASELINE.json configs[4] on one GPU: device-timed passes of the whole path."""
    import torch
    import paper_2012_06478_b200 as rms
    import rms_inputs as ri
    torch.cuda.set_device(0)
    rms.load_library()
    base = ri.make_config("cfg4", args.scale, n_walkers=1000, n_steps=args.mc_steps, n_dir=60)
    sub = base.substrate
    labels_dev = torch.from_numpy(sub.labels.view(np.int16)).cuda()
    stream = torch.cuda.current_stream()
    for n_dir in (1, 60):
        dirs = ri.fibonacci_dirs(n_dir) if n_dir > 1 else np.array([[0.0, 0.0, 1.0]])
        b = np.linspace(0.0, 25.0, 11) if n_dir > 1 else np.array([1.0])
        dt = base.sequence.dt_ms
        seq = ri.pgse_sequence(dt, args.mc_steps, 0.4 * args.mc_steps * dt, 0.6 * args.mc_steps * dt, b, dirs,
                               snap_steps=[args.mc_steps])
        layout = {"auto": rms.binding.RMS_LAYOUT_AUTO, "x": rms.binding.RMS_LAYOUT_X_FASTEST, "z": rms.binding.RMS_LAYOUT_Z_FASTEST}[args.layout]
        for lattice, flags, sflags in (("facemask", 0, layout), ("facemask, dictionary lattice", 0, layout | rms.binding.RMS_LATTICE_DICT),
                                       ("labels", rms.RMS_RUN_LABEL_GATHER, layout)):
            for n_w in (100_000, 1_000_000, 10_000_000, 100_000_000):
                if n_w > args.sweep_max_walkers:
                    continue
                reps = 3 if n_w <= 1_000_000 else 1
                rms.simulate(sub, seq, min(n_w, 1_000_000), base.seed, flags=flags, substrate_flags=sflags, device_labels=labels_dev)   # warm-up
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record(stream)
                k_ms = 0.0
                for _ in range(reps):
                    r = rms.simulate(sub, seq, n_w, base.seed, flags=flags, substrate_flags=sflags, device_labels=labels_dev)
                    k_ms += r["kernel_ms"]
                e1.record(stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / reps
                steps = float(n_w) * args.mc_steps
                print(json.dumps({"sweep": "cfg4", "walkers": n_w, "mc_steps": args.mc_steps, "directions": n_dir,
                                  "b_values": int(seq.gamp.shape[1]), "lattice_path": lattice, "layout": args.layout, "pass_ms": ms,
                                  "step_kernel_ms": k_ms / reps, "walker_steps_per_s": steps / (ms * 1e-3),
                                  "step_kernel_walker_steps_per_s": steps / (k_ms / reps * 1e-3),
                                  "issue_roofline_frac": ALGORITHMIC_INSTR_PER_STEP * steps / (k_ms / reps * 1e-3) /
                                  (N_SM * LANES_PER_SM * 1.965e9)}), flush=True)
                rms.load_library().rms_memory_trim()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.sweep:
        run_sweep(args)
        return
    import torch
    import torch.distributed as dist
    import paper_2012_06478_b200 as rms

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rms.load_library()

    cfg = make_workload(args)
    sub, seq = cfg.substrate, cfg.sequence
    n_walkers, mc_steps = args.walkers, args.mc_steps
    first_id = rank * n_walkers                       # weak scaling: every rank owns its own walker-id range
    flags = rms.RMS_RUN_LABEL_GATHER if args.lattice == "labels" else 0
    if args.fp64:
        flags |= rms.binding.RMS_RUN_FP64
    if args.no_slices:
        flags |= rms.binding.RMS_RUN_NO_SLICES
    if args.general_kernel:
        flags |= rms.binding.RMS_RUN_GENERAL_KERNEL
    flags |= {"ec": 0, "rs": rms.binding.RMS_RUN_REJECTION_SAMPLING, "erl": rms.binding.RMS_RUN_ERL}[args.interaction]
    sflags = {"auto": rms.binding.RMS_LAYOUT_AUTO, "x": rms.binding.RMS_LAYOUT_X_FASTEST, "z": rms.binding.RMS_LAYOUT_Z_FASTEST}[args.layout]
    if args.lattice_format == "dict":
        sflags |= rms.binding.RMS_LATTICE_DICT
    t_ms = np.asarray(seq.snap_steps, np.float64) * seq.dt_ms

    labels_dev = torch.from_numpy(sub.labels.view(np.int16)).cuda()          # resident in HBM before timing
    labels_pin = torch.from_numpy(sub.labels.view(np.int16)).pin_memory()    # e2e: pinned host buffer
    labels_pin_np = labels_pin.numpy().view(np.uint16)
    stream = torch.cuda.current_stream()

    sub_pin = dataclasses.replace(sub, labels=labels_pin_np)   # same substrate, labels in pinned host memory

    def one_pass(device):
        if device:   # labels already resident in HBM: adopted in place
            r = rms.simulate(sub, seq, n_walkers, cfg.seed, first_id=first_id, flags=flags, substrate_flags=sflags,
                             device_labels=labels_dev)
        else:        # host labels: rms_substrate_create copies them host -> device inside the call
            r = rms.simulate(sub_pin, seq, n_walkers, cfg.seed, first_id=first_id, flags=flags, substrate_flags=sflags)
        if world > 1:
            r = rms.api.allreduce_result(r, t_ms)
        return r

    def timed(n_iter, device):
        kernel_ms, launches = 0.0, 0
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        r = None
        for _ in range(n_iter):
            r = one_pass(device)
            kernel_ms += r["kernel_ms"]
            launches += r["n_launches"] + 2           # + neighbourhood-lattice build + walker init kernels
        e1.record(stream)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        dev_ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([dev_ms, wall * 1e3], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dev_ms, wall = float(t[0]), float(t[1]) / 1e3
        return dev_ms, wall, kernel_ms, launches, r

    timed(args.warmup, True)
    sampler = ClockSampler(local)
    sampler.start()
    dev_ms, wall, kernel_ms, launches, r = timed(args.steps, True)
    clocks = sampler.stop()
    total_steps = float(world) * n_walkers * mc_steps * args.steps
    value = total_steps / (dev_ms * 1e-3)

    e2e = None
    if not args.no_e2e:
        timed(1, False)
        e_ms, e_wall, _, _, re = timed(args.steps, False)
        h2d = sub.labels.nbytes + sub.D.nbytes + sub.T2.nbytes + sub.kappa.nbytes + sub.label_class.nbytes + \
            sub.label_allowed.nbytes + seq.wave.nbytes + seq.gamp.nbytes + seq.dirs.nbytes + seq.snap_steps.nbytes
        d2h = sum(re[k].nbytes for k in rms.api.RAW_SUMS) + 64
        e2e = {"value": total_steps / (e_ms * 1e-3), "unit": "walker-steps/s", "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": e_ms / args.steps, "wall_ms_per_step": 1e3 * e_wall / args.steps}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (rms_step_kernel): ALU issue bound
    peaks_file = ROOT / "MEASURED_PEAKS.json"
    sm_mhz = clocks.get("sm_mhz") or 1965.0
    peak_ginstr = N_SM * LANES_PER_SM * sm_mhz * 1e6 / 1e9
    k_ms_per_launch = kernel_ms / args.steps
    achieved_ginstr = ALGORITHMIC_INSTR_PER_STEP * n_walkers * mc_steps / (k_ms_per_launch * 1e-3) / 1e9
    cap = NCU_CAPTURES.get((args.substrate, args.lattice, args.layout, args.lattice_format, n_walkers, mc_steps, bool(args.fp64))) \
        if args.waves == 1 and args.interaction == "ec" and not args.no_slices and not args.general_kernel else None
    traffic = cap["bytes"] if cap else None
    roofline = {"bound": "alu", "kernel": "rms_step_fast_kernel" if args.lattice == "facemask" else "rms_step_kernel",
                "achieved": achieved_ginstr, "peak": peak_ginstr,
                "unit": "Ginstr/s (thread-instructions)", "frac": achieved_ginstr / peak_ginstr,
                "traffic": traffic, "traffic_source": cap["source"] if cap else None,
                "algorithmic_instr_per_walker_step": ALGORITHMIC_INSTR_PER_STEP, "kernel_ms_per_launch": k_ms_per_launch,
                "kernel_share_of_step": kernel_ms / dev_ms,
                "peak_source": f"148 SM x 128 lanes x SM clock measured during the run ({sm_mhz:.0f} MHz; "
                               f"MEASURED_PEAKS.json present: {peaks_file.exists()})"}

    # second roofline candidate: random-gather ceilings measured on this GPU, against the gather rate of the
    # step kernel (0.68 voxel changes per walker-step, one 8-byte octant word each)
    try:
        g_l2 = rms.binding.rms_gather_probe(48 << 20, 4, 2048)
        g_hbm = rms.binding.rms_gather_probe(2 << 30, 4, 512)
        k_rate = 0.68 * n_walkers * mc_steps / (k_ms_per_launch * 1e-3)
        k_dram = (traffic / 32.0) / (k_ms_per_launch * 1e-3) if traffic else None
        roofline["gather"] = {"kernel_gathers_per_s": k_rate, "kernel_dram_sectors_per_s": k_dram,
                              "ceiling_l2_resident_48MB": g_l2, "ceiling_hbm_2GB": g_hbm,
                              "dram_sectors_frac_of_hbm_ceiling": (k_dram / g_hbm) if k_dram else None,
                              "unit": "random 4-byte gathers/s (one 32-byte sector each); kernel_dram_sectors from the ncu capture"}
    except Exception as ex:      # the probe is a report, never a reason to lose the bench line
        roofline["gather"] = {"error": str(ex)}

    cpu_baseline = None
    if not args.no_cpu_baseline:
        import oracle
        threads = oracle.rms_oracle.default_threads()
        sample = min(args.cpu_sample_walkers, n_walkers)
        t0 = time.perf_counter()
        ro = oracle.run(sub, seq, sample, cfg.seed, first_id=0, n_threads=threads)
        dt = time.perf_counter() - t0
        cpu_baseline = {"value": sample * mc_steps / dt, "unit": "walker-steps/s", "cores": threads, "kind": "oracle",
                        "sample": f"first {sample} walker ids x {mc_steps} steps of the same workload ({dt:.1f} s)"}

    line = {"metric": "walker_steps_per_s", "value": value, "unit": "walker-steps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if args.fp64 else "f32", "data": "synthetic", "config": workload_config(args, cfg),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "wall_ms_per_step": 1e3 * wall / args.steps,
            "check": {"S_b_max_dir0": float(abs(r["S"][0, -1, 0])), "n_encounters": r["n_encounters"],
                      "n_membrane_faces": r["substrate_info"]["n_membrane_faces"],
                      "dict_entries": r["substrate_info"]["dict_entries"],
                      "dict_escaped_voxels": r["substrate_info"]["dict_escaped_voxels"]}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
