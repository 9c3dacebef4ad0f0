#!/usr/bin/env python
"""bench.py — spin-flip attempts per ns of the B200 hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole hot path over one batch of synthetic input:
sg_reset (disorder + initial state on device) -> first half of the sweeps with parallel tempering
(thermalisation) -> second half with PT and overlap measurement + accumulation.
Default workload: BASELINE.json configs[1] (C2: L=8, 2048 samples, 4 replicas, 20 temperatures,
2^14 sweeps, PT every sweep).  `value` = flip attempts of all ranks / device time (max over ranks).
N > 1: every rank simulates its own 2048-sample shard of a larger disorder pool (weak scaling,
global Philox keys, no data-path collective; one final all-reduce of the per-slot moment sums).
Prints ONE JSON line on rank 0.
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

from paper_1403_4560_b200 import workloads as W  # noqa: E402

ALU_OPS_PER_WORDSITE = 30     # algorithmic ALU-pipe lane-ops per 32-sample word-site update:
#                               6 bond XOR3 + 8 count + 7 threshold carries + 4 compare/flip + 5 Philox share
HBM_BYTES_PER_WORDSITE_LAUNCH = 8   # spin word read once + written once per LAUNCH of a resident kernel
# dram__bytes_read.sum + dram__bytes_write.sum of the roofline launch below, from the ncu --set full captures
# summarised in profiles/r01_v3_resident_kernels.md (C2) and profiles/r01_v4_final_kernels.md (C3, C5)
NCU_TRAFFIC_BYTES = {"C2": 10.92e6, "C3": 114.6e6, "C5": 8.746e9}
ALU_LANES_PER_SM = 64         # INT/LOP3 lanes per SM per clock (16 per SMSP x 4; B300_MICROARCH pipe table)
N_SM = 148


def probe_alu_peak(stream):
    """Measured ALU-pipe (LOP3) peak in lane-ops/s: bench-only micro-benchmark (csrc/probe/alu_probe.cu),
    a library of its own, not part of the product ABI."""
    import ctypes as C
    from paper_1403_4560_b200 import build
    lib = C.CDLL(build.build_probe())
    lib.sgprobe_alu_peak.restype = C.c_int
    lib.sgprobe_alu_peak.argtypes = [C.c_void_p, C.c_void_p]
    v = C.c_double()
    rc = lib.sgprobe_alu_peak(C.c_void_p(stream.cuda_stream), C.byref(v))
    if rc != 0:
        raise RuntimeError("sgprobe_alu_peak failed: %d" % rc)
    return v.value


def peaks():
    p = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            j = json.load(f)
        p.update(hbm_gbs=float(j["hbm_gbs"]), sm_max_mhz=float(j.get("sm_max_mhz", 1965.0)), src="measured")
    except Exception:
        pass
    return p


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.05)

    def result(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


def step_plan(w):
    """(n_sweeps, pt_every, meas_every) segments of one step (R16)."""
    half = w.n_sweeps // 2
    if w.meas_every:
        return [(half, w.pt_every, 0), (w.n_sweeps - half, w.pt_every, w.meas_every)]
    return [(w.n_sweeps, w.pt_every, 0)]


# ------------------------------------------------------------------------------ oracle arm
def oracle_rate(w, n_samples, n_sweeps, threads):
    """Time the CPU oracle as it stands: n_samples samples of workload w for n_sweeps sweeps with the
    workload's PT / measurement cadence, `threads` samples at a time.  Returns (attempts/ns, seconds)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import ea_oracle as O
    temps = w.temps()
    O.lib()

    def one(s):
        o = O.Oracle(w.L, w.h, w.n_replicas, temps, kind=w.kind, seed=w.seed, sample=s)
        half = n_sweeps // 2
        o.run(half, w.pt_every, 0)
        o.run(n_sweeps - half, w.pt_every, w.meas_every)
        o.close()

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(one, range(n_samples)))
    dt = time.perf_counter() - t0
    attempts = w.N * n_samples * w.n_replicas * w.n_temps * n_sweeps
    return attempts / dt / 1e9, dt


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    threads = min(cores, 32)
    per_sweep = w.N * w.n_replicas * w.n_temps * 40e-9            # ~40 ns per attempt per core
    n_sweeps = int(max(16, min(w.n_sweeps, 4.0 / per_sweep)))       # ~4 s of CPU work per sample
    n_sweeps -= n_sweeps % max(1, 2 * max(w.meas_every, 1))
    n_sweeps = max(n_sweeps, 2 * max(w.meas_every, 1))
    for _ in range(args.warmup):
        oracle_rate(w, threads, max(2, n_sweeps // 16), threads)
    rates, secs = [], []
    for _ in range(args.steps):
        r, dt = oracle_rate(w, threads, n_sweeps, threads)
        rates.append(r)
        secs.append(dt)
    total_attempts = w.N * threads * w.n_replicas * w.n_temps * n_sweeps * args.steps
    value = total_attempts / sum(secs) / 1e9
    sample = "%d samples x %d sweeps of %s per step (PT every %d, measure every %d in the 2nd half)" % (
        threads, n_sweeps, w.name, w.pt_every, w.meas_every)
    print(json.dumps({
        "impl": "reference", "metric": "spin_flip_attempts_per_ns", "value": value, "unit": "flips/ns",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": workload_config(w, args.gpus), "gpu_launches": 0,
        "cpu_baseline": {"value": value, "unit": "flips/ns", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "flips/ns", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_config(w, n_gpus):
    return {"workload": "%s: L=%d, %d samples/GPU x %d replicas x %d temperatures, %s couplings, h=%g, %d sweeps, "
                        "PT every %d, measure every %d in the 2nd half" % (
                            w.name, w.L, w.n_samples, w.n_replicas, w.n_temps, "+-J" if w.kind == W.PMJ else "Gaussian fp32",
                            w.h, w.n_sweeps, w.pt_every, w.meas_every),
            "L": w.L, "n_samples_per_gpu": w.n_samples, "n_replicas": w.n_replicas, "n_temps": w.n_temps,
            "n_sweeps": w.n_sweeps, "pt_every": w.pt_every, "meas_every": w.meas_every, "seed": w.seed,
            "parallelism": "samples sharded over %d GPU(s), no data-path collective" % n_gpus,
            "l2": "state regenerated on device every step; 256 MiB L2 flush between timed steps"}


# -------------------------------------------------------------------------------- our arm
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    from paper_1403_4560_b200 import sg, shard

    pk = peaks()
    temps = np.asarray(w.temps(), dtype=np.float64)
    stream = torch.cuda.Stream(device=dev)
    need = sg.sg_workspace_bytes(w.L, w.n_samples, w.n_replicas, w.n_temps, w.kind)
    workspace = torch.empty(need + 256, dtype=torch.uint8, device=dev)
    sim = sg.Simulation(w.L, w.h, w.n_samples, w.n_replicas, temps, w.kind, w.seed, workspace=workspace, stream=stream)
    first, _ = shard.shard_range(w.n_samples * world, world, rank)
    sim.sg_set_first_sample(first)
    plan = step_plan(w)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        sim.sg_reset()
        for seg in plan:
            sim.sg_run(*seg)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = sim.sg_get_launch_count()
    evs = []
    with torch.cuda.stream(stream):
        for _ in range(args.steps):
            flush.zero_()                                  # L2 flush, outside the events
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            step()
            e1.record(stream)
            evs.append((e0, e1))
    barrier()
    launches = sim.sg_get_launch_count() - launches0
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(step_ms))

    # dominant kernel alone (the sweep), same process and clocks: CUDA events on the library's stream around
    # each of `reps` launches of n_k back-to-back sweeps (one launch each on the resident-kernel paths)
    n_k = 256 if w.N * w.n_samples < (1 << 28) else 16
    reps = 3
    sim.sg_sweep(8)
    l0 = sim.sg_get_launch_count()
    kev = []
    for _ in range(reps):
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record(stream)
        sim.sg_sweep(n_k)
        k1.record(stream)
        kev.append((k0, k1))
    torch.cuda.synchronize(dev)
    sweep_launches = sim.sg_get_launch_count() - l0
    sweep_ms = float(sum(a.elapsed_time(b) for a, b in kev)) / reps          # per n_k sweeps
    sweep_launches //= reps
    alu_peak_measured = probe_alu_peak(stream) / 1e12                  # T lane-ops/s, LOP3 micro-benchmark
    sampler.stop_flag = True
    sampler.join()

    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms_max = float(t.item())
    attempts_per_step = w.flip_attempts() * world
    value = attempts_per_step * args.steps / (total_ms_max * 1e6)          # per ns

    # end to end through the C-ABI with host buffers: create (host temperatures -> device tables),
    # run, read the moment accumulators back into pinned host memory, destroy.
    pinned = torch.empty((w.n_samples, w.n_temps, sg.NMOM), dtype=torch.float64).pin_memory()
    pin_np = pinned.numpy()
    e2e_steps = max(1, min(args.steps, 3))
    h2d = w.n_temps * 8 + w.n_temps * 192 + 5761 * 8 + 1441 * 4 + 2 * w.L * 8
    d2h = pin_np.nbytes
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        s2 = sg.Simulation(w.L, w.h, w.n_samples, w.n_replicas, temps, w.kind, w.seed, workspace=workspace, stream=stream)
        s2.sg_set_first_sample(first)
        s2.sg_reset()
        for seg in plan:
            s2.sg_run(*seg)
        s2.sg_get_moments_into(pin_np)
        s2.close()
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_value = attempts_per_step * e2e_steps / (float(t.item()) * 1e9)

    # the one exchange step of the sharded job: disorder sums of the moment accumulators
    sums = torch.from_numpy(pin_np.sum(axis=0)).to(dev)
    if world > 1:
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)

    if rank == 0:
        wordsites_per_sweep = w.N * w.n_words * w.n_replicas * w.n_temps if w.kind == W.PMJ else w.N * w.n_samples * w.n_replicas * w.n_temps
        nominal = ALU_LANES_PER_SM * N_SM * pk["sm_max_mhz"] * 1e6 / 1e12       # T lane-ops / s
        peak = alu_peak_measured
        ach = ALU_OPS_PER_WORDSITE * wordsites_per_sweep * n_k / (sweep_ms * 1e-3) / 1e12
        sweep_rate = w.flip_attempts(n_k) / (sweep_ms * 1e6)
        launch_s = sweep_ms * 1e-3 / max(1, sweep_launches)
        hbm_ach = HBM_BYTES_PER_WORDSITE_LAUNCH * wordsites_per_sweep / launch_s / 1e9 if w.kind == W.PMJ else None
        roofline = {"bound": "alu", "kernel": "sweep (+-J multispin)", "achieved": ach, "peak": peak, "unit": "Tlaneop/s",
                    "frac": ach / peak, "traffic": NCU_TRAFFIC_BYTES.get(w.name),
                    "peak_source": "measured in this run: dependency-free LOP3 micro-benchmark (csrc/probe/alu_probe.cu); "
                                   "nominal 64 INT lanes/SM/clk x 148 SMs x %.0f MHz = %.2f" % (pk["sm_max_mhz"], nominal),
                    "peak_nominal": nominal, "frac_of_nominal": ach / nominal,
                    "alu_ops_per_wordsite": ALU_OPS_PER_WORDSITE, "launch_us": 1e6 * launch_s,
                    "launches_timed": sweep_launches * reps, "sweeps_per_launch": n_k // max(1, sweep_launches),
                    "sweep_only_flips_per_ns": sweep_rate,
                    "share_of_step": (sweep_ms / n_k) * w.n_sweeps / (total_ms / args.steps),
                    "hbm": {"achieved": hbm_ach, "peak": pk["hbm_gbs"], "unit": "GB/s",
                            "frac": (hbm_ach / pk["hbm_gbs"]) if hbm_ach else None,
                            "note": "algorithmic 8 B per word-site per LAUNCH (state resident in shared memory for all "
                                    "sweeps of a launch): HBM is not the binding roof, the ALU pipe is (DESIGN.md 6)"}}
        if w.kind != W.PMJ:
            roofline.update({"kernel": "sweep (Gaussian fp32)", "note": "no roofline target for the Gaussian path"})
        out = {"metric": "spin_flip_attempts_per_ns", "value": value, "unit": "flips/ns", "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps,
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "u32" if w.kind == W.PMJ else "f32", "data": "synthetic",
               "config": workload_config(w, world), "clocks": sampler.result(),
               "e2e": {"value": e2e_value, "unit": "flips/ns", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
               "gpu_launches": int(launches), "roofline": roofline,
               "paper_context": "33 ps/attempt = 30.3 flips/ns on a GTX 580 (PAPER.md:68); other hardware, not a target"}
        if world == 1 and not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            threads = min(cores, 32)
            per_sweep = w.N * w.n_replicas * w.n_temps * 40e-9
            n_sw = int(max(32, min(w.n_sweeps, 45.0 / per_sweep)))        # ~10-20 s of CPU work (the oracle runs ~12 ns per attempt)
            n_sw -= n_sw % 32
            r, dt = oracle_rate(w, threads, n_sw, threads)
            out["cpu_baseline"] = {"value": r, "unit": "flips/ns", "cores": threads, "kind": "oracle",
                                   "sample": "%d samples x %d sweeps of %s (same PT / measurement cadence), %.1f s" % (
                                       threads, n_sw, w.name, dt)}
        print(json.dumps(out))
    sim.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=sorted(W.BY_NAME))
    ap.add_argument("--sweeps", type=int, default=0, help="override the workload's sweep count (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    w = W.BY_NAME[args.workload]
    if args.sweeps:
        w = w.scaled(n_sweeps=args.sweeps)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
