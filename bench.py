#!/usr/bin/env python
"""bench.py -- throughput of the ensemble Cahn-Hilliard ADI step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

A "step" is one time step of the whole hot path (RHS stencil -> one cyclic-pentadiagonal sweep
per axis -> fused update, with the F/dF/dt/mass reduction at the config's sampling stride) over
the whole ensemble of the workload.  metric = grid-point updates per second.  One JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1911_03386_b200 import inputs  # noqa: E402

METRIC = "grid-point updates/sec (fp64 ensemble CH ADI step)"
UNIT = "updates/s"
FALLBACK_HBM_GBS = 6650.0       # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent

# Algorithmic bytes per grid-point update per kernel:
# every kernel reads and writes one fp64 field; the last sweep also reads C^n for the fused update.
ALGO_BYTES = {
    2: {"rhs": 16, "rhs_diag": 16, "sweep_x": 16, "sweep_y": 24,
        "rhs_sweep_y": 16, "rhs_sweep_y_diag": 16, "sweep_x_update": 24,       # fused 2D step: 40 B per update
        "step_local": 16},                                                     # one-pass local step: read C^n, write C^{n+1}
    3: {"rhs": 16, "rhs_diag": 16, "sweep_x": 16, "sweep_y": 16, "sweep_z": 24, "sweep_xy": 16},   # plane kernel: x + y in one pass
}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed
# `ncu --set full` capture (profiles/), keyed by (workload, kernel); None until captured.
# value = (bytes per launch, the committed capture it was read from).  One launch under `ncu --set full`: caches are
# flushed before the launch, so the L2 hits the live step gets from walking the ensemble up in one kernel and down in
# the next do not show, and part of the write-back is still in L2 when the launch ends.
# member-resident stepping: DFMA + DADD + DMUL per grid-point update (ncu, profiles/r02_ncu_full_resident.md) and the fp64 peak
RESIDENT_FP64_INSTR_PER_UPDATE = 30.1
ALU_PEAK_TINSTR = 148 * 64 * 1.965e9 / 1e12

NCU_TRAFFIC_BYTES = {
    ("cfg3", "sweep_x_update"): (749.5e6, "profiles/r01_v8_ncu_full_cfg3.md"),
    ("cfg3", "rhs_sweep_y"): (485.6e6, "profiles/r01_v8_ncu_full_cfg3.md"),
    ("cfg3", "step_local"): (656.1e6, "profiles/r02_ncu_full_local.md"),
}


def workload_desc(name):
    c = inputs.CONFIGS[name]
    return f"{name}: {c['D']}D {'x'.join([str(c['N'])] * c['D'])} x {c['ensemble']} members, gamma={c['gamma']}, dt={c['dt']}, stride={c['stride']}"


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------- oracle legs
def oracle_sample(name, steps, warmup=0, max_members=None):
    """Time the CPU oracle, as it stands, on a bounded sample of the workload: the first
    min(cores, ensemble) members (OpenMP over members), `steps` time steps."""
    from oracle import ch_oracle
    c = inputs.CONFIGS[name]
    cores = ch_oracle.num_threads()
    members = min(cores, c["ensemble"]) if max_members is None else min(max_members, c["ensemble"])
    C0 = inputs.config_state(name, members=range(members))
    if warmup:
        C0 = ch_oracle.step(C0, c["gamma"], c["dt"], warmup)
    t = time.perf_counter()
    ch_oracle.step(C0, c["gamma"], c["dt"], steps)
    dt = time.perf_counter() - t
    updates = members * c["N"] ** c["D"] * steps
    return {"value": updates / dt, "unit": UNIT, "cores": min(cores, members), "kind": "oracle",
            "sample": f"first {members} of {c['ensemble']} members of {name}, {steps} steps, gcc -O2 -fopenmp over members",
            "seconds": dt, "ms_per_step": dt / steps * 1e3}


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    name = args.workload
    c = inputs.CONFIGS[name]
    r = oracle_sample(name, args.steps, warmup=args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_desc(name), "note": "CPU oracle on host cores; each step is one time step of a bounded member sample"},
        "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------- CUDA arm
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def run_ours(args):
    import torch
    from paper_1911_03386_b200 import binding as B, build
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path is the only path (no CPU fallback)")
    build.build()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_1911_03386_b200 import shard

    name = args.workload
    c = inputs.CONFIGS[name]
    M, N, D, stride = c["ensemble"], c["N"], c["D"], c["stride"]
    if args.members:                 # same recipe, another ensemble size (not a BASELINE.json config then)
        M = args.members
    pts = M * N ** D
    K, W = args.steps, args.warmup

    # weak scaling: every rank steps its own full ensemble (disjoint seeds), no data-path collective
    seeds_off = rank * M
    cb = c["cbar"]
    cbars = [cb[k % len(cb)] for k in range(M)] if isinstance(cb, (list, tuple)) else [cb] * M
    host = torch.empty((M,) + (N,) * D, dtype=torch.float64).pin_memory()
    host.numpy()[...] = inputs.initial_state([c["seed0"] + seeds_off + k for k in range(M)], N, D, cbars, c["amp"])
    host_out = torch.empty_like(host).pin_memory()

    stream = torch.cuda.current_stream()
    opts = {}
    for kv in args.option:
        k, v = kv.split("=")
        opts[k] = int(v)
    ens = B.Ensemble(M, N, D, c["gamma"], c["dt"], stream=stream.cuda_stream, options=opts)
    dstate = host.to(dev, non_blocking=True)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg: inputs already in HBM when the timed region starts.
    # the K-step region is repeated `reps` times (median reported, min/max beside it).  Every
    # repetition starts at the same phase of the sampling stride, chosen so that ceil(K / stride) sampling steps (the
    # `_diag` kernel variants + k_finish, row a-5) fall inside it whatever K is; the count is read back from the
    # library (ch_series_count) and reported as `samples_in_timed_region`.
    R = max(1, args.reps)
    phase = 1 if K % stride == 0 else (stride - (K % stride) // 2) % stride
    cap = (W + (R + 1) * (K + stride)) // stride + 4
    ens.set_state(dstate)
    ens.set_series(stride, cap)
    ens.step(W)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    rep_ms, rep_samples, rep_launches = [], [], []
    for _ in range(R):
        n = B.ch_step_count(ens.ctx)
        ens.step((phase - n) % stride)          # untimed: align the region with the sampling stride
        barrier()
        l0, s0 = B.ch_launch_count(ens.ctx), B.ch_series_count(ens.ctx)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ens.step(K)
        e1.record(stream)
        barrier()
        rep_launches.append(B.ch_launch_count(ens.ctx) - l0)
        rep_samples.append(B.ch_series_count(ens.ctx) - s0)
        rep_ms.append(shard.max_over_ranks(e0.elapsed_time(e1) * 1e-3, device=dev) * 1e3)
    time.sleep(0.15)
    clocks = sampler.stop()
    order = sorted(range(R), key=lambda i: rep_ms[i])
    med = order[(R - 1) // 2]                    # the median repetition (lower median for even R)
    secs, launches, samples_in = rep_ms[med] * 1e-3, rep_launches[med], rep_samples[med]
    value = world * pts * K / secs
    repetitions = {"n": R, "ms_per_step_median": rep_ms[med] / K, "ms_per_step_min": min(rep_ms) / K,
                   "ms_per_step_max": max(rep_ms) / K, "samples_per_repetition": rep_samples}

    fuse_mode_used = B.ch_get_option(ens.ctx, "fuse_mode") if D == 2 else None
    # ---- per-kernel leg: same steps with every launch bracketed by CUDA events on the stream
    B.ch_profile(ens.ctx, 1)
    ens.set_state(dstate)
    ens.set_series(stride, cap)
    ens.step(W)
    ens.step((phase - B.ch_step_count(ens.ctx)) % stride)
    B.ch_profile_read(ens.ctx)
    ens.step(K)
    prof = B.ch_profile_read(ens.ctx)
    B.ch_profile(ens.ctx, 0)
    peak, peak_src = measured_peak()
    kernels = {}
    for kind, (ms, cnt) in prof.items():
        if cnt and kind in ALGO_BYTES[D]:
            avg = ms / cnt
            gbs = pts * ALGO_BYTES[D][kind] / (avg * 1e-3) / 1e9
            kernels[kind] = {"launches": cnt, "avg_ms": avg, "algo_bytes_per_update": ALGO_BYTES[D][kind],
                             "achieved_gbs": gbs, "frac": gbs / peak}
    if prof.get("step_resident", (0.0, 0))[1]:
        # member-resident stepping (fuse_mode 6): ONE launch runs all K steps out of shared memory, so the bound is the fp64
        # pipe, not HBM: fp64 instructions per update counted by ncu, peak from the unit count and clock
        ms, cnt = prof["step_resident"]
        tinstr = pts * K * RESIDENT_FP64_INSTR_PER_UPDATE / (ms * 1e-3) / 1e12
        kernels["step_resident"] = {"launches": cnt, "avg_ms": ms / cnt, "steps_per_launch": K,
                                    "fp64_instr_per_update": RESIDENT_FP64_INSTR_PER_UPDATE, "achieved_tinstr_s": tinstr,
                                    "frac": tinstr / ALU_PEAK_TINSTR, "hbm_bytes_per_update": 16.0 / K}
    total_kernel_ms = sum(ms for ms, _ in prof.values())
    # bytes one step must move in the pass structure that ran: fused 2D step 16 + 24 = 40 B per update
    # (DESIGN.md section 5), three-pass 2D 56 B, four-pass 3D 72 B
    fused = "sweep_x_update" in kernels
    step_bytes = 16 if "step_local" in kernels else (40 if fused else (56 if D == 2 else (56 if "sweep_xy" in kernels else 72)))
    model_bytes = 56 if D == 2 else 72
    roofline = None
    if "step_resident" not in kernels:
        main_kinds = {k: v for k, v in kernels.items() if not k.endswith("_diag")} or kernels
        dom = max(main_kinds, key=lambda k: main_kinds[k]["avg_ms"] * main_kinds[k]["launches"])
        roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
                    "frac": kernels[dom]["frac"], "traffic": NCU_TRAFFIC_BYTES.get((name, dom), (None, None))[0],
                    "traffic_source": NCU_TRAFFIC_BYTES.get((name, dom), (None, None))[1],
                    "peak_source": peak_src, "share_of_step": kernels[dom]["avg_ms"] * kernels[dom]["launches"] / total_kernel_ms,
                    "step_algo_bytes_per_update": step_bytes,
                    "step_achieved_gbs": value / world * step_bytes / 1e9,
                    "step_frac": value / world * step_bytes / 1e9 / peak,
                    "step_frac_of_8TBs_nominal": value / world * step_bytes / 1e9 / 8000.0,
                    "step_frac_of_16B_floor": value / world * 16 / 1e9 / peak,      # read C^n once, write C^{n+1} once
                    "note": ("achieved = algorithmic bytes / live CUDA-event time; a fraction above 1 means part of those bytes came from L2: "
                             "consecutive kernels walk the ensemble in opposite directions, so each finds the tail of its predecessor's "
                             "output in the 126 MB L2 (the ncu `traffic` figure is taken with caches flushed per launch)"),
                    "unfused_model_bytes_per_update": model_bytes,
                    "unfused_model_frac": value / world * model_bytes / 1e9 / peak}

    if "step_resident" in kernels:
        kr = kernels["step_resident"]
        roofline = {"bound": "alu", "kernel": "step_resident", "achieved": kr["achieved_tinstr_s"], "peak": ALU_PEAK_TINSTR,
                    "unit": "T fp64 instr/s", "frac": kr["frac"], "traffic": None, "traffic_source": None,
                    "peak_source": "148 SMs x 64 fp64 lanes per clock (ncu sm__sass_thread_inst_executed_op_dfma peak_sustained) x 1.965 GHz, DESIGN.md 5c",
                    "share_of_step": kr["avg_ms"] * kr["launches"] / total_kernel_ms,
                    "step_algo_bytes_per_update": 16.0 / K, "step_frac_of_hbm_40B_structure": value / world * 40 / 1e9 / peak,
                    "note": ("the members stay in shared memory for the whole call: HBM traffic is 16 B / K per update, and the fraction of "
                             "the HBM roofline of the 40 B two-kernel structure this throughput would need is given for context (may exceed 1)")}

    # ---- paper-regime leg: same shape, gamma' = 66.4, dt' = 7.97 (sigma = 529, the
    # paper's gamma = 0.01, dx = 2 pi / 512, dt = 0.0012 in h = 1 units): the closure tables do not decay
    paper_regime = None
    if args.paper_regime:
        ens2 = B.Ensemble(M, N, D, 66.4, 7.97, stream=stream.cuda_stream, options=opts if "fuse" not in opts else {})
        ens2.set_state(dstate)
        ens2.set_series(stride, cap)
        ens2.step(W)
        barrier()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record(stream)
        ens2.step(K)
        p1.record(stream)
        barrier()
        psecs = shard.max_over_ranks(p0.elapsed_time(p1) * 1e-3, device=dev)
        paper_regime = {"gamma": 66.4, "dt": 7.97, "sigma": 66.4 * 7.97, "ms_per_step": psecs / K * 1e3,
                        "value": world * pts * K / psecs, "unit": UNIT,
                        "closure_chunks_K": B.ch_get_option(ens2.ctx, "K"), "fuse_mode": B.ch_get_option(ens2.ctx, "fuse_mode")}
        ens2.close()

    # ---- end-to-end leg: the user's job through the C ABI with HOST buffers (pinned):
    # ch_set_state(host) -> ch_step(K) with the series -> series D2H + ch_energy(host) + ch_get_state(host)
    series_host = torch.empty((cap, M, 4), dtype=torch.float64).pin_memory()
    eout = np.empty((M, 4), dtype=np.float64)
    barrier()
    ens.set_series(stride, cap)
    B.ch_run_host(ens.ctx, host.numpy(), host_out.numpy(), 3)       # warm-up: creates the three internal streams
    barrier()
    t0 = time.perf_counter()
    ens.set_series(stride, cap)
    B.ch_run_host(ens.ctx, host.numpy(), host_out.numpy(), K)       # H2D, K steps (with sampling), D2H, chunk-pipelined
    B.ch_energy(ens.ctx, eout)
    ns = B.ch_series_count(ens.ctx)
    series_host[:ns].copy_(ens._series[:ns], non_blocking=True)
    barrier()
    e2e_secs = shard.max_over_ranks(time.perf_counter() - t0, device=dev)
    state_bytes = pts * 8
    e2e = {"value": world * pts * K / e2e_secs, "unit": UNIT,
           "h2d_bytes_per_step": state_bytes / K, "d2h_bytes_per_step": (state_bytes + ns * M * 32 + M * 32) / K,
           "seconds": e2e_secs, "job": f"ch_run_host(host {state_bytes >> 20} MiB in, {K} steps, {state_bytes >> 20} MiB out; member chunks pipelined over 3 streams) + series/energy to host"}
    assert np.isfinite(eout).all() and np.isfinite(host_out.numpy()).all()

    ens.close()
    if rank == 0:
        if args.no_cpu_baseline:      # profiling runs (ncu) only: skip the CPU leg
            cpu = {"value": None, "unit": UNIT, "cores": 0, "kind": "oracle", "sample": "skipped (--no-cpu-baseline)"}
        else:
            cpu = oracle_sample(name, max(5, int(1.5e8 / N ** D)))    # ~10-20 s of CPU work per core
            one = oracle_sample(name, max(2, int(3e7 / N ** D)), max_members=1)   # one member on one thread, a few seconds
            cpu["value_1thread"] = one["value"]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": secs / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_desc(name) + (f" [--members {M}]" if args.members else ""), "members_per_gpu": M, "options": opts, "fuse_mode": fuse_mode_used, "parallelism": f"ensemble-sharded x{world} (no data-path collective)",
                       "l2": (f"working set {2 * state_bytes >> 20} MiB per GPU, larger than the 126 MB L2; no explicit flush" if 2 * state_bytes > (126 << 20)
                              else f"working set {2 * state_bytes >> 20} MiB per GPU: SMALLER than the 126 MB L2 and not flushed (a small-ensemble parity config, not the headline)"),
                       "sampling": (f"F, dF/dt, beta, mass every {stride} steps; {samples_in} sampling step(s) inside the {K}-step timed region "
                                    f"(every repetition starts at step n = {phase} mod {stride})")},
            "samples_in_timed_region": samples_in, "repetitions": repetitions,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "kernels": kernels, "paper_regime": paper_regime,
            "cpu_baseline": {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "value_1thread") if k in cpu},
        }
        print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", default="cfg3", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--reps", type=int, default=5, help="repetitions of the timed K-step region (median reported)")
    ap.add_argument("--option", action="append", default=[], metavar="KEY=INT",
                    help="kernel-variant option passed to ch_set_option (include/ch.h), e.g. fuse=5; repeatable")
    ap.add_argument("--members", type=int, default=0, help="override the ensemble size of the workload (same recipe and seeds)")
    ap.add_argument("--no-paper-regime", dest="paper_regime", action="store_false",
                    help="skip the extra timed leg at the paper's gamma dt / h^4 = 529")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (for runs under ncu)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
