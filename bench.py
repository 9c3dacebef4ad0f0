#!/usr/bin/env python
"""bench.py — spin-flip attempts per ns of the B200 hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole hot path over one batch of synthetic input:
sg_reset (disorder + initial state on device) -> the config's sweeps with parallel tempering at its cadence
(first half = thermalisation; second half with overlap measurement + accumulation where the
config measures).  Default workload: BASELINE.json configs[4] (C5: L=32, 8192 samples, 4 replicas,
32 temperatures, 1024 sweeps, PT every 4) — the largest single-GPU config, the one north_star calls the
throughput run.  `value` = flip attempts of all ranks / device time (max over ranks).  The same JSON line
carries short runs of the other +-J configs and of the Gaussian one (`other_configs`).
N > 1: every rank simulates its own shard of a larger disorder pool (weak scaling, global Philox keys, no
data-path collective; one final all-reduce of the per-slot moment / energy sums).  Prints ONE JSON line on rank 0.
"""
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

from paper_1403_4560_b200 import workloads as W  # noqa: E402

# Algorithmic ALU-pipe lane-ops per 32-sample word-site update, by the comparison the kernels of the
# context actually run (sg_get_accept_variant): 6 bond XOR3 + 8 count + threshold carries + 4 compare/flip + 5 Philox share
#   binary search (h != 0): 3 carries -> 26;  carry chain (h = 0): 7 carries -> 30;  general select: not modelled (30 assumed)
ALU_OPS_BY_VARIANT = {2: 26, 1: 30, 0: 30}
VARIANT_NAME = {2: "binary-search compare (3 carries)", 1: "carry chain (7 carries)", 0: "general 14-mask select (not modelled; 30 assumed)"}
HBM_BYTES_PER_WORDSITE_LAUNCH = 8   # spin word read once + written once per LAUNCH of a resident kernel
# What `ncu --set full` reported for ONE roofline launch (the sweep kernel alone, n_k sweeps) of each +-J config, from the
# capture summarised in the file named beside it: dram bytes (read + write), ALU-pipe active fraction
# (sm__pipe_alu_cycles_active / sm__cycles_active) and executed thread-instructions per word-site (all pipes / ALU pipe
# only).  Pointers to profiles/, not re-measured by this run; the line says so.  `frac` (algorithmic ops / peak) must stay
# below `pipe_alu_active` (executed ops / peak) of the same launch: useful work cannot exceed executed work.
NCU_CAPTURE = {
    "C2": {"traffic": 10.90e6, "pipe_alu_active": 0.6890, "pipe_alu_elapsed": 0.6091, "inst_per_wordsite": 50.0,
           "alu_inst_per_wordsite": 28.6, "source": "profiles/r03_kernels.md (k_ladder8_pmj<4,1,0>, 256 plain sweeps)"},
    "C3": {"traffic": 114.7e6, "pipe_alu_active": 0.6880, "pipe_alu_elapsed": 0.6784, "inst_per_wordsite": 55.1,
           "alu_inst_per_wordsite": 30.5, "source": "profiles/r03_kernels.md (k_ladder_pmj<12,1,0>, 256 plain sweeps)"},
    "C5": {"traffic": 8.759e9, "pipe_alu_active": 0.6611, "pipe_alu_elapsed": 0.6589, "inst_per_wordsite": 48.4,
           "alu_inst_per_wordsite": 27.7, "source": "profiles/r03_kernels.md (k_res32_pmj<1>, 16 sweeps)"},
}
# Gaussian path (C4), k_gladder<16>, one 256-sweep launch: executed thread instructions per flip attempt, issue-slot and pipe
# utilisation, dram bytes of the launch
GAUSS_CAPTURE = {"C4": {"inst_per_flip": 60.4, "issue_active": 0.776, "pipe_alu_active": 0.567, "pipe_fma_active": 0.413,
                        "traffic": 514.6e6, "source": "profiles/r03_kernels.md (k_gladder<16>, 256 plain sweeps)"}}
ALU_LANES_PER_SM = 64         # INT/LOP3 lanes per SM per clock (16 per SMSP x 4; B300_MICROARCH pipe table)
N_SM = 148


def probe_alu_peak(stream):
    """Measured ALU-pipe (LOP3) peak in lane-ops/s: bench-only micro-benchmark (bench_probe/alu_probe.cu),
    a library of its own beside bench.py, not part of the product package or its ABI."""
    import ctypes as C
    from bench_probe import build as probe_build
    lib = C.CDLL(probe_build.build_probe())
    lib.sgprobe_alu_peak.restype = C.c_int
    lib.sgprobe_alu_peak.argtypes = [C.c_void_p, C.c_void_p]
    v = C.c_double()
    rc = lib.sgprobe_alu_peak(C.c_void_p(stream.cuda_stream), C.byref(v))
    if rc != 0:
        raise RuntimeError("sgprobe_alu_peak failed: %d" % rc)
    return v.value


def peaks():
    p = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback (B200_PROFILING.md)"}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            j = json.load(f)
        p.update(hbm_gbs=float(j["hbm_gbs"]), sm_max_mhz=float(j.get("sm_max_mhz", 1965.0)), src="MEASURED_PEAKS.json")
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
    per_sweep = w.N * w.n_replicas * w.n_temps * 15e-9            # ~15 ns per attempt per core
    n_sweeps = int(max(8, min(w.n_sweeps, 4.0 / per_sweep)))        # ~4 s of CPU work per sample
    q = max(1, 2 * max(w.meas_every, 1), 2 * w.pt_every)
    n_sweeps = max(q, n_sweeps - n_sweeps % q)
    for _ in range(args.warmup):
        oracle_rate(w, threads, max(2, n_sweeps // 16), threads)
    secs = []
    for _ in range(args.steps):
        _, dt = oracle_rate(w, threads, n_sweeps, threads)
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
                        "PT every %d, %s" % (
                            w.name, w.L, w.n_samples, w.n_replicas, w.n_temps, "+-J" if w.kind == W.PMJ else "Gaussian fp32",
                            w.h, w.n_sweeps, w.pt_every,
                            ("measure every %d in the 2nd half" % w.meas_every) if w.meas_every else
                            "no measurement inside the step (R16)"),
            "L": w.L, "n_samples_per_gpu": w.n_samples, "n_replicas": w.n_replicas, "n_temps": w.n_temps,
            "n_sweeps": w.n_sweeps, "pt_every": w.pt_every, "meas_every": w.meas_every, "seed": w.seed,
            "parallelism": "samples sharded over %d GPU(s), no data-path collective" % n_gpus,
            "l2": "state regenerated on device every step; 256 MiB L2 flush between timed steps"}


# -------------------------------------------------------------------------------- our arm
def wordsites_per_sweep(w):
    if w.kind == W.PMJ:
        return w.N * w.n_words * w.n_replicas * w.n_temps
    return w.N * w.n_samples * w.n_replicas * w.n_temps


def time_steps(sim, w, plan, steps, warmup, stream, flush, barrier):
    """W untimed + K timed steps; returns (per-step ms list, launches in the timed steps)."""
    import torch

    def step():
        sim.sg_reset()
        for seg in plan:
            sim.sg_run(*seg)

    for _ in range(warmup):
        step()
    barrier()
    launches0 = sim.sg_get_launch_count()
    evs = []
    with torch.cuda.stream(stream):
        for _ in range(steps):
            flush.zero_()                                  # L2 flush, outside the events
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            step()
            e1.record(stream)
            evs.append((e0, e1))
    barrier()
    return [a.elapsed_time(b) for a, b in evs], sim.sg_get_launch_count() - launches0


def time_sweep_kernel(sim, w, stream, dev, reps=3):
    """The dominant kernel alone (the sweep), same process and clocks: CUDA events on the library's stream around each
    of `reps` launches of n_k back-to-back sweeps.  Returns (ms per n_k sweeps, n_k, launches per n_k sweeps)."""
    import torch
    n_k = 256 if w.N * w.n_samples < (1 << 28) else 16
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
    launches = (sim.sg_get_launch_count() - l0) // reps
    return float(sum(a.elapsed_time(b) for a, b in kev)) / reps, n_k, launches


def roofline_block(w, sweep_ms, n_k, sweep_launches, step_ms, alu_peak, pk, variant=2):
    ws = wordsites_per_sweep(w)
    nominal = ALU_LANES_PER_SM * N_SM * pk["sm_max_mhz"] * 1e6 / 1e12       # T lane-ops / s
    sweep_rate = w.flip_attempts(n_k) / (sweep_ms * 1e6)
    launch_s = sweep_ms * 1e-3 / max(1, sweep_launches)
    share = (sweep_ms / n_k) * w.n_sweeps / step_ms
    if w.kind != W.PMJ:
        # Gaussian byte/fp32 path: bound by instruction ISSUE (ncu: issue slots 78 % busy, ALU pipe 57 %, FMA pipe 41 %, LSU 16 %,
        # no memory stall; profiles/r03_kernels.md).  Peak = 4 warp instructions per clock per SM = 128 thread-instruction slots.
        # The work figure is the EXECUTED thread-instruction count per flip attempt of the named capture (no smaller
        # algorithmic count is claimed for this path), so frac is an issue-slot utilisation, not an algorithmic efficiency.
        cap = GAUSS_CAPTURE.get(w.name)
        peak = 128.0 * N_SM * pk["sm_max_mhz"] * 1e6 / 1e12
        ach = cap["inst_per_flip"] * sweep_rate * 1e9 / 1e12 if cap else None
        return {"bound": "issue", "kernel": "sweep (Gaussian fp32 byte path, k_gladder)", "achieved": ach, "peak": peak,
                "unit": "Tinst/s", "frac": ach / peak if cap else None, "traffic": cap["traffic"] if cap else None,
                "peak_source": "nominal: 4 schedulers x 1 warp instruction (32 threads) per clock x 148 SMs x %.0f MHz" % pk["sm_max_mhz"],
                "inst_per_flip_attempt": cap["inst_per_flip"] if cap else None,
                "ncu": dict(cap, note="from the named `ncu --set full` capture of one 256-sweep launch (a pointer to profiles/, not "
                                      "re-measured by this run)") if cap else None,
                "sweep_only_flips_per_ns": sweep_rate, "share_of_step": share,
                "launch_us": 1e6 * launch_s, "sweeps_per_launch": n_k // max(1, sweep_launches),
                "note": "BASELINE.json sets no roofline target for the Gaussian path (parity only); executed-instruction "
                        "fraction of the issue-slot peak"}
    ops = ALU_OPS_BY_VARIANT[variant]
    ach = ops * ws * n_k / (sweep_ms * 1e-3) / 1e12
    hbm_ach = HBM_BYTES_PER_WORDSITE_LAUNCH * ws / launch_s / 1e9
    cap = NCU_CAPTURE.get(w.name, {})
    return {"bound": "alu", "kernel": "sweep (+-J multispin)", "achieved": ach, "peak": alu_peak, "unit": "Tlaneop/s",
            "frac": ach / alu_peak, "traffic": cap.get("traffic"),
            "accept_variant": VARIANT_NAME[variant],
            "ncu": {"pipe_alu_active": cap.get("pipe_alu_active"), "pipe_alu_elapsed": cap.get("pipe_alu_elapsed"),
                    "inst_per_wordsite": cap.get("inst_per_wordsite"),
                    "alu_inst_per_wordsite": cap.get("alu_inst_per_wordsite"), "source": cap.get("source"),
                    "note": "from the named `ncu --set full` capture of one such launch (a pointer to profiles/, not "
                            "re-measured by this run): sm__pipe_alu_cycles_active as a fraction of active / of elapsed SM "
                            "cycles, executed thread instructions and ALU-pipe lane slots per word-site.  frac counts "
                            "algorithmic ops over wall time, so it must stay below pipe_alu_elapsed"},
            "peak_source": "measured in this run: dependency-free LOP3 micro-benchmark (bench_probe/alu_probe.cu); "
                           "nominal 64 INT lanes/SM/clk x 148 SMs x %.0f MHz = %.2f" % (pk["sm_max_mhz"], nominal),
            "peak_nominal": nominal, "frac_of_nominal": ach / nominal,
            "alu_ops_per_wordsite": ops, "launch_us": 1e6 * launch_s,
            "sweeps_per_launch": n_k // max(1, sweep_launches),
            "sweep_only_flips_per_ns": sweep_rate, "share_of_step": share,
            "hbm": {"achieved": hbm_ach, "peak": pk["hbm_gbs"], "peak_source": pk["src"], "unit": "GB/s", "frac": hbm_ach / pk["hbm_gbs"],
                    "note": "algorithmic 8 B per word-site per LAUNCH (state resident in shared memory for all "
                            "sweeps of a launch): HBM is not the binding roof, the ALU pipe is (DESIGN.md 6)"}}


def short_run(sg, torch, name, sweeps, dev, stream, flush, alu_peak, pk):
    """A short run of another config for the `other_configs` block: whole-step value (same cadence, fewer sweeps),
    sweep kernel alone, roofline fraction."""
    w = W.BY_NAME[name].scaled(n_sweeps=sweeps)
    temps = np.asarray(w.temps(), dtype=np.float64)
    sim = sg.Simulation(w.L, w.h, w.n_samples, w.n_replicas, temps, w.kind, w.seed, stream=stream)

    def barrier():
        torch.cuda.synchronize(dev)

    ms, launches = time_steps(sim, w, step_plan(w), 3, 1, stream, flush, barrier)
    step_ms = float(np.mean(ms))
    sweep_ms, n_k, sl = time_sweep_kernel(sim, w, stream, dev)
    prop, acc = sim.sg_get_pt_stats()
    variant = sim.sg_get_accept_variant() if w.kind == W.PMJ else 0
    sim.close()
    rb = roofline_block(w, sweep_ms, n_k, sl, step_ms, alu_peak, pk, variant)
    out = {"workload": "%s at %d of %d sweeps (same PT / measurement cadence)" % (name, sweeps, W.BY_NAME[name].n_sweeps),
           "value": w.flip_attempts() / (step_ms * 1e6), "unit": "flips/ns", "ms_per_step": step_ms,
           "ms_per_step_best": float(np.min(ms)), "ms_per_step_median": float(np.median(ms)),
           "sweep_only_flips_per_ns": rb["sweep_only_flips_per_ns"], "frac": rb["frac"],
           "alu_ops_per_wordsite": rb.get("alu_ops_per_wordsite"), "accept_variant": rb.get("accept_variant"),
           "pipe_alu_active": (rb.get("ncu") or {}).get("pipe_alu_active"),
           "pipe_alu_elapsed": (rb.get("ncu") or {}).get("pipe_alu_elapsed"), "ncu_source": (rb.get("ncu") or {}).get("source"),
           "gpu_launches_per_step": launches // 3,
           "pt_acceptance": float(acc.sum()) / max(1.0, float(prop.sum()))}
    if w.kind == W.PMJ and w.n_samples % 32:
        # idle lanes of the last packed word are simulated too (report both rates)
        all_lanes = 32.0 * w.n_words / w.n_samples
        out["active_lanes"] = "%d of %d" % (w.n_samples, 32 * w.n_words)
        out["value_all_lanes"] = out["value"] * all_lanes
        out["sweep_only_flips_per_ns_all_lanes"] = out["sweep_only_flips_per_ns"] * all_lanes
    return out


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

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank)
    sampler.start()
    step_ms, launches = time_steps(sim, w, plan, args.steps, args.warmup, stream, flush, barrier)
    total_ms = float(sum(step_ms))
    sweep_ms, n_k, sweep_launches = time_sweep_kernel(sim, w, stream, dev)
    prop, acc = sim.sg_get_pt_stats()
    variant = sim.sg_get_accept_variant() if w.kind == W.PMJ else 0
    # the launches the step really uses (sweeps between two exchanges + the exchange work fused into them), timed alone:
    # 64 sweeps at the workload's PT cadence, no measurement
    cad_ms = cad_launches = None
    if w.pt_every > 0:
        sim.sg_run(4 * w.pt_every, w.pt_every, 0)
        l0 = sim.sg_get_launch_count()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        sim.sg_run(64, w.pt_every, 0)
        c1.record(stream)
        torch.cuda.synchronize(dev)
        cad_ms, cad_launches = float(c0.elapsed_time(c1)), int(sim.sg_get_launch_count() - l0)
    sampler.stop_flag = True
    sampler.join()
    alu_peak_measured = probe_alu_peak(stream) / 1e12                        # T lane-ops/s, LOP3 micro-benchmark
    sim.close()

    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms_max = float(t.item())
    attempts_per_step = w.flip_attempts() * world
    value = attempts_per_step * args.steps / (total_ms_max * 1e6)          # per ns

    # end to end through the C-ABI with host buffers: create (host temperatures -> device tables), run, read the
    # step's result back into pinned host memory (moment accumulators where the config measures, else the per-system
    # energies (U, M) the run ended with), destroy.
    measures = w.meas_every > 0
    if measures:
        pinned = torch.empty((w.n_samples, w.n_temps, sg.NMOM), dtype=torch.float64).pin_memory()
        pin_np = pinned.numpy()
        d2h = pin_np.nbytes
    else:
        pinU = torch.empty((w.n_samples, w.n_replicas, w.n_temps), dtype=torch.int64).pin_memory()
        pinM = torch.empty((w.n_samples, w.n_replicas, w.n_temps), dtype=torch.int32).pin_memory()
        d2h = pinU.numpy().nbytes + pinM.numpy().nbytes
    e2e_steps = max(1, min(args.steps, 3))
    h2d = w.n_temps * 8 + w.n_temps * 192 + 5761 * 8 + 1441 * 4 + 2 * w.L * 8
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        s2 = sg.Simulation(w.L, w.h, w.n_samples, w.n_replicas, temps, w.kind, w.seed, workspace=workspace, stream=stream)
        s2.sg_set_first_sample(first)
        s2.sg_reset()
        for seg in plan:
            s2.sg_run(*seg)
        if measures:
            s2.sg_get_moments_into(pin_np)
        else:
            s2.sg_get_energies_cached_into(pinU.numpy(), pinM.numpy())
        s2.close()
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_value = attempts_per_step * e2e_steps / (float(t.item()) * 1e9)

    # the one exchange step of the sharded job: disorder sums over ALL ranks' samples of what the
    # step returned; reported so that the reduction is exercised and checkable (N = 1: the local sums)
    if measures:
        local = torch.from_numpy(pin_np.sum(axis=0)).to(dev)                 # [n_temps][NMOM]
    else:
        local = torch.stack([torch.from_numpy(pinU.numpy().sum(axis=(0, 1)).astype(np.float64)),
                             torch.from_numpy(pinM.numpy().sum(axis=(0, 1)).astype(np.float64))]).to(dev)
    sums = shard.reduce_moment_sums(local)
    n_sys = float(w.n_samples * world * w.n_replicas)
    if measures:
        n_meas = (w.n_sweeps - w.n_sweeps // 2) // w.meas_every
        n_terms = float(w.n_samples * world * n_meas * (w.n_replicas * (w.n_replicas - 1) // 2))
        reduced = {"what": "[<q^2>] per slot over all ranks' samples, pairs and measurements (accumulator 1 / terms)",
                   "per_slot": [float(x) / n_terms for x in sums[:, 1].tolist()]}
    else:
        reduced = {"what": "mean energy per spin (2U - 3N - hM)/N per slot over all ranks' samples and replicas",
                   "per_slot": [float((2.0 * u / n_sys - 3.0 * w.N - w.h * m / n_sys) / w.N) for u, m in zip(sums[0].tolist(), sums[1].tolist())]}

    if rank == 0:
        ms_per_step = total_ms_max / args.steps
        roofline = roofline_block(w, sweep_ms, n_k, sweep_launches, total_ms / args.steps, alu_peak_measured, pk, variant)
        if cad_ms is not None:
            roofline["step_cadence"] = {
                "what": "64 sweeps with PT every %d through sg_run, no measurement: the launches the timed step is made of" % w.pt_every,
                "flips_per_ns": w.flip_attempts(64) / (cad_ms * 1e6), "launches": cad_launches,
                "launch_us": 1e3 * cad_ms / max(1, cad_launches)}
        out = {"metric": "spin_flip_attempts_per_ns", "value": value, "unit": "flips/ns", "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
               "ms_per_step_best": float(np.min(step_ms)), "ms_per_step_median": float(np.median(step_ms)),
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "u32" if w.kind == W.PMJ else "f32", "data": "synthetic",
               "config": workload_config(w, world), "clocks": sampler.result(),
               "e2e": {"value": e2e_value, "unit": "flips/ns", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "h2d_note": "computed from the sizes of the tables sg_create uploads (temperatures, per-slot thresholds, "
                                   "exp tables, twiddles), not counted by the library; couplings and spins are generated on the device",
                       "result": "moment accumulators" if measures else "per-system energies (U, M) of the final state"},
               "gpu_launches": int(launches), "roofline": roofline,
               "pt": {"proposed": int(prop.sum()), "accepted": int(acc.sum()),
                      "acceptance_per_pair": [round(float(a) / max(1.0, float(p)), 4) for p, a in zip(prop.tolist(), acc.tolist())]},
               "reduced_over_ranks": reduced,
               "paper_context": "33 ps/attempt = 30.3 flips/ns on a GTX 580 (PAPER.md:68); other hardware, not a target"}
        if world == 1 and not args.no_other_configs:
            others = {}
            del workspace
            torch.cuda.empty_cache()
            for name, sweeps in (("C1", 1000), ("C2", 2048), ("C3", 1024), ("C4", 256)):
                if name != w.name:
                    others[name] = short_run(sg, torch, name, sweeps, dev, stream, flush, alu_peak_measured, pk)
            out["other_configs"] = others
        if world == 1 and not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            threads = min(cores, 32)
            per_sweep = w.N * w.n_replicas * w.n_temps * 15e-9
            n_sw = int(max(8, min(w.n_sweeps, 15.0 / per_sweep)))          # ~10-20 s of CPU work (the oracle runs ~12-15 ns per attempt)
            q = max(1, 2 * max(w.meas_every, 1), 2 * w.pt_every)
            n_sw = max(q, n_sw - n_sw % q)
            r, dt = oracle_rate(w, threads, n_sw, threads)
            out["cpu_baseline"] = {"value": r, "unit": "flips/ns", "cores": threads, "kind": "oracle",
                                   "sample": "%d samples x %d sweeps of %s (same PT / measurement cadence), %.1f s" % (
                                       threads, n_sw, w.name, dt)}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5", choices=sorted(W.BY_NAME))
    ap.add_argument("--sweeps", type=int, default=0, help="override the workload's sweep count (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    args = ap.parse_args()
    world_env = os.environ.get("WORLD_SIZE")
    if args.gpus > 1 and world_env is None:
        # launched directly with --gpus N: re-run under torch.distributed.run, one rank per GPU
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%s" % (args.gpus, world_env))
    w = W.BY_NAME[args.workload]
    if args.sweeps:
        w = w.scaled(n_sweeps=args.sweeps)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
