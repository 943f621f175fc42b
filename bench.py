#!/usr/bin/env python
"""bench.py -- potential solves/s of the FFT-convolution path on synthetic disks (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A step = one pass of the whole hot path (rows a2, a3+a4r, a4phi of DESIGN.md) over one batch of
the config's synthetic density, device resident (PG_MEM_DEVICE).  Default workload: config 5
(2048x2048, the grid BASELINE.json's metric and north_star's 60 % target are quoted on).
Successive steps rotate through R distinct (Sigma, Phi) buffer pairs whose total size exceeds the
126 MB L2, so inputs do not stay cached between timed iterations.  One JSON line on stdout.

Multi-GPU (torchrun): the path does not shard ("replicas only"): every rank
runs the same workload on its own GPU, no data-path collective; value = all ranks' solves / max time.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on this box's host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2409_02294_b200.workloads import CONFIGS, make_rho3, make_sigma  # noqa: E402
from paper_2409_02294_b200 import replicas  # noqa: E402

METRIC = "potential solves/sec (fp64 FFT-convolution, log-polar thin disk)"
UNIT = "solves/s"
L2_BYTES = 126e6


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.path = tempfile.mktemp(prefix="pg_clocks_", suffix=".csv")
        self.proc = None
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        try:
            for line in open(self.path):
                t = [x.strip() for x in line.split(",")]
                if len(t) < 9:
                    continue
                try:
                    sm.append(float(t[1])); mx.append(float(t[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), t[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


dist_env = replicas.dist_env

REL_L2, MAX_REL = 1e-10, 1e-9           # north_star's parity bar (same figures as tests/test_gpu_parity.py)
REPEATS = 5                              # the K-step region is timed this many times; the median is reported


HASHED_SOURCES = ("fft.cuh", "kernels.cuh", "polargrav.cu")


def device_code_hash() -> str:
    """sha256 over the sources that decide what the three solve kernels are and how they are launched -- csrc/fft.cuh,
    csrc/kernels.cuh and csrc/polargrav.cu (grid and shared-memory sizes, lane policy, PDL attributes live there): an
    ncu record applies to the build being timed only if it was captured from the same sources."""
    import hashlib
    h = hashlib.sha256()
    for f in HASHED_SOURCES:
        with open(os.path.join(ROOT, "paper_2409_02294_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_record(cfg: int):
    """profiles/ncu_head.json: DRAM traffic and FP64 instruction counts per launch from the committed
    `ncu --set full` capture, with the commit and device-code hash it was taken at.  Returned only when that
    hash equals the hash of the sources this run was built from; otherwise the JSON line carries null and says why."""
    path = os.path.join(ROOT, "profiles", "ncu_head.json")
    if not os.path.exists(path):
        return None, "profiles/ncu_head.json not found"
    with open(path) as f:
        rec = json.load(f)
    if rec.get("device_code_sha256_16") != device_code_hash():
        return None, (f"profiles/ncu_head.json was captured at commit {rec.get('commit')} from other kernels "
                      f"(hash {rec.get('device_code_sha256_16')} != {device_code_hash()}): not reported")
    per_cfg = rec.get("configs", {}).get(str(cfg))
    if per_cfg is None:
        return None, f"profiles/ncu_head.json has no capture of config {cfg}"
    return {"commit": rec.get("commit"), "command": rec.get("command"), **per_cfg}, None


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def host_placement(gpu_index: int) -> dict:
    """Where the bench process runs relative to the GPU (section 2.3: up to +220 % on the far socket)."""
    out = {"cpu_affinity": None, "numa_node_of_process": None, "numa_node_of_gpu": None}
    try:
        cpus = sorted(os.sched_getaffinity(0))
        out["cpu_affinity"] = f"{len(cpus)} cpus: {cpus[0]}-{cpus[-1]}" if cpus else None
        cpu = cpus[0] if cpus else 0
        for node in sorted(os.listdir("/sys/devices/system/node")):
            if node.startswith("node") and os.path.exists(f"/sys/devices/system/node/{node}/cpu{cpu}"):
                out["numa_node_of_process"] = int(node[4:])
                break
    except Exception:
        pass
    try:
        bus = subprocess.run(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=pci.bus_id", "--format=csv,noheader"],
                             capture_output=True, text=True, timeout=10).stdout.strip().lower()
        if bus:
            bus = bus[-12:] if len(bus) > 12 else bus            # 00000000:1B:00.0 -> 0000:1b:00.0
            with open(f"/sys/bus/pci/devices/{bus}/numa_node") as f:
                out["numa_node_of_gpu"] = int(f.read().strip())
    except Exception:
        pass
    return out


# ------------------------------------------------------------------ CPU oracle legs
def oracle_rings(cfg: int, n: int):
    """O1 on n seeded target rings of field 0 of config `cfg` (the parity gate of the bench line)."""
    import oracle
    c = CONFIGS[cfg]
    r, phi, _, _ = oracle.grid(c.n_r, c.n_phi, c.r_in, c.r_out)
    sigma = make_sigma(cfg, r, phi)
    rng = np.random.default_rng(1)
    rings = np.unique(np.concatenate([[0, c.n_r // 2, c.n_r - 1], rng.choice(c.n_r, size=min(c.n_r, n), replace=False)])).astype(np.int32)
    return rings, oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma, rings)


def oracle_sample(cfg: int, seconds_target: float = 12.0):
    """Times oracle.potential_o1_rings on a bounded sample of target rings of config `cfg`.
    Returns (solves/s extrapolated to the whole grid, cores, description, seconds)."""
    import oracle
    c = CONFIGS[cfg]
    r, phi, _, _ = oracle.grid(c.n_r, c.n_phi, c.r_in, c.r_out)
    sigma = make_sigma(cfg, r, phi)
    cores = oracle.num_threads()
    rng = np.random.default_rng(0)
    probe = np.sort(rng.choice(c.n_r, size=min(c.n_r, cores), replace=False)).astype(np.int32)
    t0 = time.perf_counter()
    oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma, probe)
    t_probe = time.perf_counter() - t0
    waves = int(max(1, min(c.n_r // max(1, len(probe)), round(seconds_target / max(t_probe, 1e-3)))))
    rings = np.sort(rng.choice(c.n_r, size=min(c.n_r, waves * len(probe)), replace=False)).astype(np.int32)
    t0 = time.perf_counter()
    ref = oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma, rings)
    t = time.perf_counter() - t0
    frac = len(rings) / c.n_r
    solves_per_s = frac / t
    desc = (f"oracle O1 (ring-pair direct sum, gcc -O3 -march=native -fopenmp) on {len(rings)} of {c.n_r} "
            f"target rings of config {cfg} field 0 ({t:.2f} s), extrapolated to the whole grid by rings")
    return solves_per_s, cores, desc, t, rings, sigma, ref


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import oracle
    cfg = args.config
    c = CONFIGS[cfg]
    sps, cores, desc, t_one, rings, sigma, _ = oracle_sample(cfg, seconds_target=6.0)
    for _ in range(args.warmup):
        pass  # the sample above already warmed caches/threads; the oracle has no other state
    times = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        oracle.potential_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, sigma, rings)
        times.append(time.perf_counter() - t0)
    t = float(np.mean(times))
    value = (len(rings) / c.n_r) * c.batch / t / c.batch   # solves/s of one field, extrapolated
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg) + (f" -- OVERRIDDEN: batch {c.batch} (--batch; not a BASELINE.json workload)" if args.batch else ""),
                   "n_r": c.n_r, "n_phi": c.n_phi, "batch": c.batch,
                   "step": f"O1 direct sum over {len(rings)} of {c.n_r} target rings (bounded sample)"},
        "cells_per_s": value * c.n_r * c.n_phi,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "cpu": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def fp64_block(n, ms_per_launch, clocks):
    """Secondary roofline of the dominant kernel: FP64 thread instructions per second against the
    pipe's issue peak 64 x SMs x SM clock (what actually bounds cols_kernel).
    n = FP64 thread instructions per launch from profiles/ncu_head.json (None when no valid record)."""
    if n is None or ms_per_launch <= 0:
        return None
    import torch
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    mhz = (clocks or {}).get("sm_mhz") or 1965.0
    peak = FP64_LANES_PER_CLK_PER_SM * sms * mhz * 1e6
    achieved = n / (ms_per_launch * 1e-3)
    return {"bound": "alu", "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "T fp64 thread-instr/s",
            "frac": achieved / peak, "thread_instructions_per_launch": n,
            "peak_source": f"64 lanes/clk/SM x {sms} SMs x {mhz:.0f} MHz"}


def workload_name(cfg: int) -> str:
    c = CONFIGS[cfg]
    return f"BASELINE.json configs[{cfg - 1}]: {c.name}, r in [{c.r_in:g},{c.r_out:g}], eps={c.eps:g}, batch {c.batch}"


# ------------------------------------------------------------------ the CUDA path
def measure_ours(args):
    """The main line (2-D path, BASELINE.json's metric) as a dict, and the exit code of its parity gate; prints nothing."""
    import torch
    from paper_2409_02294_b200 import binding as pg, build as pg_build

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if not os.path.exists(pg.LIB_PATH):
        pg_build.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg = args.config
    c = CONFIGS[cfg]
    if args.batch:
        # NOT a BASELINE.json workload: the grid of config `cfg` with `--batch` independent fields per call, so that every
        # launch runs tens of waves (used for the steady-state ncu capture of profiles/r2_06)
        import dataclasses
        c = dataclasses.replace(c, batch=args.batch)
    field_bytes = 8 * c.n_r * c.n_phi
    pair_bytes = 2 * field_bytes * c.batch
    R = int(min(64, max(4, -(-4 * L2_BYTES // pair_bytes))))

    st = torch.cuda.Stream()
    torch.cuda.synchronize()
    t_create = time.perf_counter()
    solver = pg.Solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, max_batch=c.batch, device=local_rank,
                       cuda_stream=st.cuda_stream)
    t_create = time.perf_counter() - t_create       # tables, workspaces and row a1 (the Green's-kernel spectrum), once
    h = solver.h
    # the densities of the timed loop are resident in HBM and complete before the loop starts
    pg.pg_set_option(h, pg.PG_OPT_DENSITY_STABLE, 1)
    # the solves of the timed loop are independent (distinct resident buffer pairs): two in flight (PG_OPT_LANES),
    # joined into the timing stream by pg_flush before the end event.  Off for the host-bound small grids.
    # Grids of up to 512 x 512 take the fused single-launch path (PG_OPT_FUSED, on by default) and are bound by the
    # host's launch rate: four lanes keep four of those launches in flight.
    small = c.n_r <= 512 and c.n_phi <= 512
    lanes = args.lanes if args.lanes else (2 if c.n_r * c.n_phi >= 1 << 20 else (4 if small else 1))
    pg.pg_set_option(h, pg.PG_OPT_LANES, lanes)
    if args.no_fused:
        pg.pg_set_option(h, pg.PG_OPT_FUSED, 0)
    fused = small and not args.no_fused
    r, phi, _ = solver.grid()
    n_fields = R * c.batch
    distinct = min(n_fields, 8 if c.n_r * c.n_phi >= 1 << 22 else 32)
    base = [make_sigma(cfg, r, phi, b) for b in range(distinct)]
    host_fields = [base[k] if k < distinct else np.roll(base[k % distinct], 97 * (k // distinct), axis=1)
                   for k in range(n_fields)]
    d_sig = [torch.from_numpy(np.stack(host_fields[p * c.batch:(p + 1) * c.batch])).cuda() for p in range(R)]
    d_phi = [torch.empty_like(d_sig[p]) for p in range(R)]
    torch.cuda.synchronize()

    def step(k):
        p = k % R
        pg.pg_set_density(h, d_sig[p], c.batch, pg.PG_MEM_DEVICE)
        pg.pg_potential(h, d_phi[p], c.batch, pg.PG_MEM_DEVICE)

    def barrier():
        replicas.barrier(world)

    def max_over_ranks(x: float) -> float:
        return replicas.max_over_ranks(x, world, "cuda")

    for k in range(args.warmup):
        step(k)
    pg.pg_synchronize(h)

    # ---- timed region: exactly K steps between CUDA events on the solver's stream
    # The region of exactly K steps is timed REPEATS times (barrier + synchronize on both sides of each); the
    # median of the repeats is the reported figure, min and max go beside it (median of 5).
    sampler = ClockSampler(local_rank) if rank == 0 else None
    rep_ms = []
    n0 = pg.pg_launch_count(h)
    for _ in range(REPEATS):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier(); torch.cuda.synchronize()
        e0.record(st)
        for k in range(args.steps):
            step(k)
        pg.pg_flush(h)
        e1.record(st)
        torch.cuda.synchronize(); barrier()
        rep_ms.append(max_over_ranks(e0.elapsed_time(e1)))
    n1 = pg.pg_launch_count(h)
    ms_total = float(np.median(rep_ms))
    gate_field = d_phi[0][0].cpu().numpy() if rank == 0 else None     # field 0 as the timed region left it
    # keep the GPU busy a little longer so that short runs still collect clock samples under load
    if sampler is not None:
        t_end = time.perf_counter() + 0.6
        k = 0
        while time.perf_counter() < t_end:
            step(k); k += 1
            if k % 64 == 0:
                pg.pg_synchronize(h)
        pg.pg_synchronize(h)
    clocks = sampler.stop() if sampler is not None else None
    # ---- parity gate ("parity gate before any timing counts"): the potential of field 0 as the timed
    # loop left it in HBM, against oracle O1 on seeded rings.  Steps k = 0 (mod R) solve field 0 into d_phi[0].
    parity = {"ok": True, "what": "rank 0 only"}
    if rank == 0:
        gate_rings, gate_ref = oracle_rings(cfg, 12 if c.n_r >= 1024 else 32)
        gate_got = gate_field[gate_rings]
        gate_l2 = float(np.linalg.norm(gate_got - gate_ref) / np.linalg.norm(gate_ref))
        gate_mx = float(np.abs(gate_got / gate_ref - 1.0).max())
        parity = {"rel_l2": gate_l2, "max_rel": gate_mx, "rings": int(len(gate_rings)),
                  "bar": {"rel_l2": REL_L2, "max_rel": MAX_REL},
                  "what": "d_phi of field 0 as the timed region left it vs oracle O1 (ring-pair direct sum) on seeded rings",
                  "ok": bool(gate_l2 <= REL_L2 and gate_mx <= MAX_REL)}
    ms_per_step = ms_total / args.steps
    value = world * c.batch * 1e3 / ms_per_step
    n_launch = int(round((n1 - n0) / REPEATS)) * world

    # ---- the same K-step region with ONE solve in flight (PG_OPT_LANES = 1): what a time series gets whose step k + 1
    # depends on step k (a disk code that evolves Sigma with Phi), SURVEY 8(d)'s "one stream" protocol
    ms_one_lane = ms_per_step
    if lanes >= 2:
        pg.pg_set_option(h, pg.PG_OPT_LANES, 1)
        one = []
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier(); torch.cuda.synchronize()
            e0.record(st)
            for k in range(args.steps):
                step(k)
            e1.record(st)
            torch.cuda.synchronize(); barrier()
            one.append(max_over_ranks(e0.elapsed_time(e1)))
        ms_one_lane = float(np.median(one)) / args.steps
        pg.pg_set_option(h, pg.PG_OPT_LANES, lanes)

    # ---- per-kernel durations (events around every kernel, separate pass) -> roofline of the dominant kernel
    pg.pg_profile(h, True)
    for k in range(args.steps):
        step(k)
    kms, kn = pg.pg_kernel_times(h)
    pg.pg_profile(h, False)
    per_launch_ms = [kms[i] / max(1, kn[i]) for i in range(pg.PG_NUM_KERNELS)]
    dom = int(np.argmax(per_launch_ms))
    peak, peak_src = load_peaks()
    ncu, ncu_why = ncu_record(cfg) if not args.batch else (None, "--batch overrides the config the ncu record was captured at")
    kbytes = [pg.pg_kernel_algorithmic_bytes(h, i, c.batch) for i in range(pg.PG_NUM_KERNELS)]
    achieved = kbytes[dom] / (per_launch_ms[dom] * 1e-3) / 1e9
    # the bytes the kernel has to move as built: the column kernel reads Khat as its symmetric half (8 N_r M_h bytes less)
    needed = kbytes[dom] - (8.0 * c.n_r * (c.n_phi // 2 + 1) if dom == 1 else 0.0)
    path_bytes = pg.pg_algorithmic_bytes(h, c.batch)
    path_gbs = path_bytes / (ms_per_step * 1e-3) / 1e9

    # ---- L2-flushed variant: every step timed on its own with a >L2 memset in between (one solve at a time: the
    # lanes of PG_OPT_LANES are not ordered behind the flush on the timing stream, so they are switched off here)
    pg.pg_set_option(h, pg.PG_OPT_LANES, 1)
    flush = torch.empty(int(3 * L2_BYTES), dtype=torch.uint8, device="cuda")
    fl = []
    with torch.cuda.stream(st):
        for k in range(min(args.steps, 50)):
            flush.fill_(k & 0xFF)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st); step(k); b.record(st)
            fl.append((a, b))
    torch.cuda.synchronize()
    ms_flushed = float(np.median([a.elapsed_time(b) for a, b in fl]))
    del flush

    # ---- end to end through the C ABI with host buffers (copies inside the timed region)
    pin_in = [pg.PinnedArray((c.batch, c.n_r, c.n_phi)) for _ in range(2)]
    pin_out = [pg.PinnedArray((c.batch, c.n_r, c.n_phi)) for _ in range(2)]
    for q in range(2):
        pin_in[q].array[...] = np.stack(host_fields[q * c.batch:(q + 1) * c.batch])

    def e2e_step(k):
        q = k & 1
        pg.pg_set_density(h, pin_in[q].ptr, c.batch, pg.PG_MEM_HOST_PINNED)
        pg.pg_potential(h, pin_out[q].ptr, c.batch, pg.PG_MEM_HOST_PINNED)

    e2e_steps = max(3, min(args.steps, 40))
    for k in range(3):
        e2e_step(k)
    pg.pg_synchronize(h)
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        e2e_step(k)
    pg.pg_synchronize(h)
    t_e2e = max_over_ranks(time.perf_counter() - t0)
    e2e_value = world * c.batch * e2e_steps / t_e2e
    # serial variant: one blocking pageable-host call pair per step (PG_MEM_HOST)
    pageable_in = np.stack(host_fields[:c.batch]); pageable_out = np.empty_like(pageable_in)
    pg.pg_set_density(h, pageable_in, c.batch, pg.PG_MEM_HOST); pg.pg_potential(h, pageable_out, c.batch, pg.PG_MEM_HOST)
    t0 = time.perf_counter()
    n_pg = max(2, min(e2e_steps, 10))
    for _ in range(n_pg):
        pg.pg_set_density(h, pageable_in, c.batch, pg.PG_MEM_HOST)
        pg.pg_potential(h, pageable_out, c.batch, pg.PG_MEM_HOST)
    t_pageable = (time.perf_counter() - t0) / n_pg
    sane = bool(np.isfinite(pageable_out).all() and (pageable_out < 0).all())

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "ms_per_step_one_lane": ms_one_lane,
        "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg) + (f" -- OVERRIDDEN: batch {c.batch} (--batch; not a BASELINE.json workload)" if args.batch else ""),
                   "n_r": c.n_r, "n_phi": c.n_phi, "batch": c.batch,
                   "parallelism": "replicas only (no collective)" if world > 1 else "single GPU",
                   "path": ("one cooperative launch per solve (fused_solve_kernel: a2 | grid barrier | a3+a4r | grid barrier | a4phi)"
                            if fused else "three launches per solve (rows_fwd, cols, rows_inv) chained by programmatic dependent launch"),
                   "options": "PG_OPT_DENSITY_STABLE (densities resident and complete before the timed loop)"
                              + (f", PG_OPT_LANES={lanes} (independent solves, {lanes} in flight; pg_flush before the end event)" if lanes >= 2 else ""),
                   "l2": f"inputs larger than L2: steps rotate over {R} distinct (Sigma,Phi) buffer pairs, "
                         f"{R * pair_bytes / 1e6:.0f} MB in total vs 126 MB L2"},
        "cells_per_s": value * c.n_r * c.n_phi,
        "create_ms": 1e3 * t_create,                # pg_create_ex incl. the one-time Green's-kernel precompute (row a1); not in `value`
        "gpu_launches": n_launch,
        "repeats": {"n": REPEATS, "ms_per_step_median": ms_per_step, "ms_per_step_min": min(rep_ms) / args.steps,
                    "ms_per_step_max": max(rep_ms) / args.steps},
        "parity": parity,
        "host": host_placement(local_rank),
        "roofline": {
            "bound": "hbm", "kernel": pg.KERNEL_NAMES[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak, "frac_needed_bytes": needed / (per_launch_ms[dom] * 1e-3) / 1e9 / peak,
            "needed_bytes_per_launch": needed, "traffic": (ncu or {}).get("dram_bytes_per_launch", [None] * 3)[dom],
            "traffic_source": (f"profiles/ncu_head.json, ncu --set full at commit {ncu['commit']}" if ncu else ncu_why),
            "peak_source": peak_src,
            "algorithmic_bytes_per_launch": kbytes[dom], "ms_per_launch": per_launch_ms[dom],
            "algorithmic_bytes_note": "SURVEY.md 8(d)'s figures (56 B/cell; the 49.0 us target derives from them). The column "
                                      "kernel reads Khat as its symmetric half, so it needs 8 N_r M_h bytes less than counted here "
                                      "(84.0 instead of 100.8 MB at 2048^2); DRAM traffic per launch is in `traffic`.",
            "kernels": {pg.KERNEL_NAMES[i]: {"ms": per_launch_ms[i], "alg_bytes": kbytes[i],
                                            "gbs": kbytes[i] / (per_launch_ms[i] * 1e-3) / 1e9 if per_launch_ms[i] > 0 else None}
                        for i in range(pg.PG_NUM_KERNELS)},
            "path": {"alg_bytes_per_step": path_bytes, "gbs": path_gbs, "frac_of_peak": path_gbs / peak,
                     "frac_of_8TBs_nominal": path_gbs / 8000.0},
            "fp64": fp64_block((ncu or {}).get("fp64_thread_instructions_per_launch", [None] * 3)[dom], per_launch_ms[dom], clocks),
            "one_lane": {"ms_per_step": ms_one_lane, "gbs": path_bytes / (ms_one_lane * 1e-3) / 1e9,
                         "frac_of_peak": path_bytes / (ms_one_lane * 1e-3) / 1e9 / peak,
                         "frac_of_8TBs_nominal": path_bytes / (ms_one_lane * 1e-3) / 1e9 / 8000.0},
            "l2_flushed_one_lane_serialised": {
                "ms_per_step": ms_flushed, "frac_of_peak": path_bytes / (ms_flushed * 1e-3) / 1e9 / peak,
                "note": "one solve at a time, each timed on its own behind a > L2 memset: NOT comparable with ms_per_step "
                        "(no overlap between solves, cold L2 for Khat and the tables); compare with one_lane"},
        },
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": field_bytes * c.batch,
                "d2h_bytes_per_step": field_bytes * c.batch,
                "how": "pg_set_density + pg_potential with PG_MEM_HOST_PINNED buffers (pg_host_alloc), wall clock over "
                       f"{e2e_steps} steps, pg_synchronize at the end",
                "pageable_blocking_ms_per_step": 1e3 * t_pageable, "output_sane": sane},
        "clocks": clocks,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sps, cores, desc, _, _, _, _ = oracle_sample(cfg)
        line["cpu_baseline"] = {"value": sps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "cpu": cpu_model()}
    for a in pin_in + pin_out:
        a.free()
    solver.close()
    if small and rank == 0:
        line["batched"] = batched_small(cfg, st, args)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return line, (0 if parity["ok"] else 3)


def compact(line):
    """The figures of a secondary line that the main line carries in its `others` block."""
    rf = line.get("roofline", {})
    path = rf.get("path", {})
    par = line.get("parity", {})
    return {"workload": line["config"]["workload"], "steps": line["steps"], "ms_per_step": line["ms_per_step"],
            "value": line["value"], "unit": line["unit"], "cells_per_s": line.get("cells_per_s"),
            "gpu_launches": line.get("gpu_launches"),
            "parity": {k: par.get(k) for k in ("rel_l2", "max_rel", "ok", "what")},
            "path_gbs": path.get("gbs", rf.get("achieved")),
            "path_frac_of_peak": path.get("frac_of_peak", rf.get("frac")),
            "path_frac_of_8TBs_nominal": path.get("frac_of_8TBs_nominal", (rf.get("achieved") or 0.0) / 8000.0),
            "clocks_sm_mhz": (line.get("clocks") or {}).get("sm_mhz")}


def others_block(args):
    """Driver-witnessed figures for the workloads the default line is NOT quoted on: config 4 (8 x 1024^2), one 128^3
    Cartesian mesh level (NEXT-2) and four nested 64^3 levels (NEXT-3), 20 steps each with their own parity gates, same
    protocol as their own modes (--config 4, --cart 128, --nested 4 --cart 64), no oracle timing."""
    import copy
    out, rc = {}, 0
    for key, kw, fn in (("config4", dict(config=4), measure_ours), ("cart128", dict(cart=128), measure_cart),
                        ("nested4x64", dict(nested=4, cart=64), measure_nested)):
        a = copy.copy(args)
        a.steps, a.warmup, a.no_cpu_baseline, a.lanes, a.batch = 20, 3, True, 0, 0
        for k, v in kw.items():
            setattr(a, k, v)
        try:
            line, r = fn(a)
            out[key] = compact(line)
            rc = rc or r
        except Exception as e:                      # a secondary figure must not take the headline down with it
            out[key] = {"error": f"{type(e).__name__}: {e}"}
    return out, rc


def run_ours(args):
    line, rc = measure_ours(args)
    rank, _, world = dist_env()
    if rank == 0 and world == 1 and args.config == 5 and not args.batch and not args.no_others:
        line["others"], rc_o = others_block(args)
        rc = rc or rc_o
    if rank == 0:
        print(json.dumps(line), flush=True)
    if rc:
        sys.stderr.write(f"bench.py: PARITY GATE FAILED: {line['parity']} / others {json.dumps({k: v.get('parity', v) for k, v in line.get('others', {}).items()})}; the timing above does not count\n")
    return rc


def batched_small(cfg, st, args):
    """Configs 1-3 are single solves and bound by the host's launch rate.  The same C-ABI calls take a batch: 32
    independent fields per pg_set_density / pg_potential pair, one launch set for all of them."""
    import torch
    from paper_2409_02294_b200 import binding as pg
    c = CONFIGS[cfg]
    B = 32
    s = pg.Solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, max_batch=B, device=torch.cuda.current_device(), cuda_stream=st.cuda_stream)
    try:
        pg.pg_set_option(s.h, pg.PG_OPT_DENSITY_STABLE, 1)
        if args.no_fused:
            pg.pg_set_option(s.h, pg.PG_OPT_FUSED, 0)
        r, phi, _ = s.grid()
        base = np.stack([make_sigma(cfg, r, phi, b % 4) for b in range(B)])
        R = int(min(16, max(2, -(-4 * L2_BYTES // (2 * base.nbytes)))))
        d_sig = [torch.from_numpy(np.roll(base, 7 * p, axis=2)).cuda() for p in range(R)]
        d_phi = [torch.empty_like(x) for x in d_sig]
        torch.cuda.synchronize()
        steps = max(args.steps, 20)
        ms = []
        n0 = pg.pg_launch_count(s.h)
        for rep in range(REPEATS + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(st)
            for k in range(steps):
                pg.pg_set_density(s.h, d_sig[k % R], B, pg.PG_MEM_DEVICE)
                pg.pg_potential(s.h, d_phi[k % R], B, pg.PG_MEM_DEVICE)
            e1.record(st)
            torch.cuda.synchronize()
            if rep:
                ms.append(e0.elapsed_time(e1) / steps)
        launches = (pg.pg_launch_count(s.h) - n0) / ((REPEATS + 1) * steps)
        med = float(np.median(ms))
        # un-batched, but one host call for the whole series: pg_potential_series over the B fields of a buffer, one
        # solve (one fused launch) per field, four lanes
        pg.pg_set_option(s.h, pg.PG_OPT_LANES, 4)
        field = c.n_r * c.n_phi
        ser = []
        for rep in range(REPEATS + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(st)
            for k in range(steps):
                pg.pg_potential_series(s.h, d_sig[k % R], d_phi[k % R], B, field)
            pg.pg_flush(s.h)
            e1.record(st)
            torch.cuda.synchronize()
            if rep:
                ser.append(e0.elapsed_time(e1) / (steps * B))
        ser_med = float(np.median(ser))
        return {"batch": B, "ms_per_batch": med, "solves_per_s": B * 1e3 / med, "launches_per_batch": launches,
                "what": f"{B} independent fields per pg_set_density / pg_potential pair (resident), median of {REPEATS} repeats of {steps} batches",
                "series": {"ms_per_solve": ser_med, "solves_per_s": 1e3 / ser_med,
                           "what": f"pg_potential_series: {B} single-field solves per host call, one launch set each, PG_OPT_LANES = 4, "
                                   f"median of {REPEATS} repeats of {steps} calls"}}
    finally:
        s.close()


FP64_LANES_PER_CLK_PER_SM = 64


def run_accel(args):
    """--accel: the NEXT-4 variant kernels at the config's grid (default config 5): pg_acceleration (a_r, a_phi of the
    density last set: one forward row pass, then per component one complex column pass cols_cplx_kernel and one inverse
    row pass) and pg_potential under PG_SOFT_SOURCE (complex spectrum, one component).  Same protocol as the main line:
    resident buffers rotated beyond L2, median of REPEATS repeats of the K-step region, parity gate against
    oracle/polar_oracle_ext.c on seeded rings.  Algorithmic bytes per acceleration call (cells N = n_r n_phi, spectrum
    S = 16 n_r (n_phi/2 + 1) bytes): row forward 8 N + S; per component the column pass reads S, reads the complex kernel
    spectrum 2 S and writes S, the inverse row pass reads S and writes 8 N  ->  24 N + 11 S."""
    import torch
    import oracle
    from paper_2409_02294_b200 import binding as pg, build as pg_build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if not os.path.exists(pg.LIB_PATH):
        pg_build.build()
    cfg = args.config
    c = CONFIGS[cfg]
    st = torch.cuda.Stream()
    solver = pg.Solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, device=0, cuda_stream=st.cuda_stream)
    h = solver.h
    r, phi, _ = solver.grid()
    field_bytes = 8 * c.n_r * c.n_phi
    R = int(min(32, max(4, -(-4 * L2_BYTES // (3 * field_bytes)))))
    base = [make_sigma(cfg, r, phi, b) for b in range(min(R, 4))]
    d_sig = [torch.from_numpy(np.roll(base[k % len(base)], 97 * (k // len(base)), axis=1)).cuda() for k in range(R)]
    d_ar = [torch.empty_like(d_sig[0]) for _ in range(R)]
    d_ap = [torch.empty_like(d_sig[0]) for _ in range(R)]
    torch.cuda.synchronize()
    peak, peak_src = load_peaks()
    spec = 16.0 * c.n_r * (c.n_phi // 2 + 1)
    out = {}

    def timed(step, steps):
        for k in range(max(3, args.warmup)):
            step(k)
        pg.pg_synchronize(h)
        rep = []
        for _ in range(REPEATS):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(st)
            for k in range(steps):
                step(k)
            e1.record(st)
            torch.cuda.synchronize()
            rep.append(e0.elapsed_time(e1) / steps)
        return float(np.median(rep)), min(rep), max(rep)

    def acc_step(k):
        pg.pg_set_density(h, d_sig[k % R], 1, pg.PG_MEM_DEVICE)
        pg.pg_acceleration(h, d_ar[k % R], d_ap[k % R], 1, pg.PG_MEM_DEVICE)

    def phi_step(k):
        pg.pg_set_density(h, d_sig[k % R], 1, pg.PG_MEM_DEVICE)
        pg.pg_potential(h, d_ar[k % R], 1, pg.PG_MEM_DEVICE)

    sampler = ClockSampler(0)
    steps = max(1, args.steps)
    rc = 0
    rings = np.unique(np.random.default_rng(5).integers(0, c.n_r, 6 if c.n_r >= 1024 else 16)).astype(np.int32)
    for soft, name in ((pg.PG_SOFT_SYMMETRIC, "symmetric"), (pg.PG_SOFT_SOURCE, "source")):
        pg.pg_set_softening(h, soft)
        ms, lo, hi = timed(acc_step, steps)
        n0 = pg.pg_launch_count(h)
        acc_step(0)
        launches = pg.pg_launch_count(h) - n0
        alg = 24.0 * c.n_r * c.n_phi + 11.0 * spec
        gbs = alg / (ms * 1e-3) / 1e9
        # parity: field 0 as the timed loop left it
        ref_phi, ref_r, ref_p = oracle.ext_o1_rings(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, soft, base[0], rings)
        g_r, g_p = d_ar[0].cpu().numpy()[rings], d_ap[0].cpu().numpy()[rings]
        mag = np.hypot(ref_r, ref_p)
        l2 = max(float(np.linalg.norm(g - q) / np.linalg.norm(q)) for g, q in ((g_r, ref_r), (g_p, ref_p)))
        mx = max(float((np.abs(g - q) / mag).max()) for g, q in ((g_r, ref_r), (g_p, ref_p)))
        ok = bool(l2 <= REL_L2 and mx <= MAX_REL)
        rc = rc or (0 if ok else 3)
        out[f"acceleration_{name}"] = {"ms_per_step": ms, "ms_min": lo, "ms_max": hi, "launches_per_step": launches,
                                       "algorithmic_bytes_per_step": alg, "gbs": gbs, "frac_of_peak": gbs / peak,
                                       "parity": {"rel_l2": l2, "max_rel_to_magnitude": mx, "rings": int(len(rings)), "ok": ok}}
        if soft != pg.PG_SOFT_SYMMETRIC:
            ms, lo, hi = timed(phi_step, steps)
            alg = 16.0 * c.n_r * c.n_phi + 6.0 * spec          # rows 8 N + S; column pass S + 2 S + S; inverse rows S + 8 N
            gbs = alg / (ms * 1e-3) / 1e9
            got = d_ar[0].cpu().numpy()[rings]
            l2 = float(np.linalg.norm(got - ref_phi) / np.linalg.norm(ref_phi)); mx = float(np.abs(got / ref_phi - 1).max())
            ok = bool(l2 <= REL_L2 and mx <= MAX_REL)
            rc = rc or (0 if ok else 3)
            out[f"potential_{name}"] = {"ms_per_step": ms, "ms_min": lo, "ms_max": hi, "algorithmic_bytes_per_step": alg, "gbs": gbs,
                                        "frac_of_peak": gbs / peak, "parity": {"rel_l2": l2, "max_rel": mx, "rings": int(len(rings)), "ok": ok}}
    clocks = sampler.stop()
    a = out["acceleration_source"]
    line = {"metric": "acceleration solves/sec (fp64 FFT convolution, a_r and a_phi of one field; row NEXT-4)", "value": 1e3 / a["ms_per_step"],
            "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": max(3, args.warmup), "ms_per_step": a["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg) + " -- pg_acceleration, PG_SOFT_SOURCE (equal to -grad Phi)", "n_r": c.n_r, "n_phi": c.n_phi,
                       "l2": f"inputs larger than L2: steps rotate over {R} (Sigma, a_r, a_phi) buffer triples"},
            "parity": a["parity"],
            "roofline": {"bound": "hbm", "kernel": "whole call (rows_fwd, 2 x cols_cplx, 2 x rows_inv)", "achieved": a["gbs"], "peak": peak,
                         "unit": "GB/s", "frac": a["frac_of_peak"], "traffic": None, "peak_source": peak_src,
                         "algorithmic_bytes_per_step": a["algorithmic_bytes_per_step"]},
            "variants": out, "clocks": clocks}
    solver.close()
    print(json.dumps(line), flush=True)
    if rc:
        sys.stderr.write("bench.py: PARITY GATE FAILED in --accel\n")
    return rc


def run_direct(args):
    """--direct: times the on-GPU cross-check (row a5, direct_kernel: tiled all-pairs summation from the
    coordinates) on one field of the config and reports pair interactions per second.  Not the headline
    metric and never a fallback; FP64-pipe bound."""
    import torch
    from paper_2409_02294_b200 import binding as pg, build as pg_build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if not os.path.exists(pg.LIB_PATH):
        pg_build.build()
    c = CONFIGS[args.config]
    st = torch.cuda.Stream()
    solver = pg.Solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, device=0, cuda_stream=st.cuda_stream)
    r, phi, _ = solver.grid()
    d_s = torch.from_numpy(make_sigma(args.config, r, phi, 0)).cuda()
    d_p = torch.empty_like(d_s)
    torch.cuda.synchronize()
    rings = min(c.n_r, 888 if c.n_r * c.n_phi > 1 << 20 else c.n_r)     # bounded: two full waves of target rings (3 CTAs per SM)
    steps = max(1, min(args.steps, 5))

    def step():
        pg.pg_set_density(solver.h, d_s, 1, pg.PG_MEM_DEVICE)
        pg.pg_potential_direct_rings(solver.h, d_p, 0, rings, pg.PG_MEM_DEVICE)

    step(); pg.pg_synchronize(solver.h)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(steps):
        step()
    e1.record(st)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    pairs = float(rings) * c.n_phi * c.n_r * c.n_phi
    line = {"metric": "pair interactions/sec (fp64 direct summation cross-check, row a5)", "value": pairs / (ms * 1e-3),
            "unit": "pairs/s", "n_gpus": 1, "steps": steps, "warmup": 1, "ms_per_step": ms, "higher_is_better": True,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "target_rings": rings, "pairs_per_step": pairs},
            "extrapolated_full_grid_s": ms * 1e-3 * c.n_r / rings}
    solver.close()
    print(json.dumps(line), flush=True)
    return 0


def run_staging(args):
    """--staging: row a6's own measurement.  The paper times the host-to-device
    transfer of one 128^3 array: about 1 ms from pinned memory, about 3 ms from pageable memory (A100 40 GB, PCIe).
    Here the same 16.8 MB (128^3 fp64 = a 1024 x 2048 grid) goes through the library's own staging calls,
    PG_MEM_HOST (pageable: memcpy into the owned pinned buffer, then cudaMemcpyAsync) against PG_MEM_HOST_PINNED
    (cudaMemcpyAsync straight from the caller's pinned buffer), upload and download separately; then the batch
    pipeline of config 4 (8 fields): upload-only, solve-only, download-only and all three overlapped."""
    import torch
    from paper_2409_02294_b200 import binding as pg, build as pg_build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if not os.path.exists(pg.LIB_PATH):
        pg_build.build()
    reps = max(5, min(args.steps, 30))

    def med(f, n=reps):
        ts = []
        for _ in range(n):
            t0 = time.perf_counter(); f(); ts.append(time.perf_counter() - t0)
        return 1e3 * float(np.median(ts))

    st = torch.cuda.Stream()
    n_r, n_phi = 1024, 2048                                  # 2^21 cells = 128^3
    s = pg.Solver(n_r, n_phi, 1.0, 1000.0, 0.01, device=0, cuda_stream=st.cuda_stream)
    h = s.h
    from paper_2409_02294_b200.workloads import random_sigma
    sig = random_sigma(n_r, n_phi, 1)
    pin_in, pin_out = pg.PinnedArray((n_r, n_phi)), pg.PinnedArray((n_r, n_phi))
    pin_in.array[...] = sig
    page_in, page_out = sig.copy(), np.empty_like(sig)
    d_sig = torch.from_numpy(sig).cuda(); d_phi = torch.empty_like(d_sig)
    nbytes = sig.nbytes

    def up(mem, buf):
        pg.pg_set_density(h, buf, 1, mem); pg.pg_synchronize(h)

    def solve_dev():
        pg.pg_set_density(h, d_sig, 1, pg.PG_MEM_DEVICE); pg.pg_potential(h, d_phi, 1, pg.PG_MEM_DEVICE); pg.pg_synchronize(h)

    def solve_to(mem, buf):
        pg.pg_set_density(h, d_sig, 1, pg.PG_MEM_DEVICE); pg.pg_potential(h, buf, 1, mem); pg.pg_synchronize(h)

    for _ in range(3):
        up(pg.PG_MEM_HOST_PINNED, pin_in.ptr); up(pg.PG_MEM_HOST, page_in); solve_dev()
        solve_to(pg.PG_MEM_HOST_PINNED, pin_out.ptr); solve_to(pg.PG_MEM_HOST, page_out)
    h2d_pinned = med(lambda: up(pg.PG_MEM_HOST_PINNED, pin_in.ptr))
    h2d_pageable = med(lambda: up(pg.PG_MEM_HOST, page_in))
    t_solve = med(solve_dev)
    d2h_pinned = med(lambda: solve_to(pg.PG_MEM_HOST_PINNED, pin_out.ptr)) - t_solve
    d2h_pageable = med(lambda: solve_to(pg.PG_MEM_HOST, page_out)) - t_solve
    ok = bool(np.array_equal(pin_out.array, page_out) and (page_out < 0).all())
    pin_in.free(); pin_out.free(); s.close()

    # ---- the batch pipeline of config 4: H2D(b+1) || solve(b) || D2H(b-1)
    c = CONFIGS[4]
    s = pg.Solver(c.n_r, c.n_phi, c.r_in, c.r_out, c.eps, max_batch=c.batch, device=0, cuda_stream=st.cuda_stream)
    h = s.h
    shape = (c.batch, c.n_r, c.n_phi)
    pin_in, pin_out = pg.PinnedArray(shape), pg.PinnedArray(shape)
    r, phi, _ = s.grid()
    pin_in.array[...] = np.stack([make_sigma(4, r, phi, b) for b in range(c.batch)])
    d_b = torch.from_numpy(pin_in.array.copy()).cuda(); d_o = torch.empty_like(d_b)

    def b_up():
        pg.pg_set_density(h, pin_in.ptr, c.batch, pg.PG_MEM_HOST_PINNED); pg.pg_synchronize(h)

    def b_solve():
        pg.pg_set_density(h, d_b, c.batch, pg.PG_MEM_DEVICE); pg.pg_potential(h, d_o, c.batch, pg.PG_MEM_DEVICE); pg.pg_synchronize(h)

    def b_down():
        pg.pg_set_density(h, d_b, c.batch, pg.PG_MEM_DEVICE); pg.pg_potential(h, pin_out.ptr, c.batch, pg.PG_MEM_HOST_PINNED); pg.pg_synchronize(h)

    def b_all(n=6):
        for _ in range(n):
            pg.pg_set_density(h, pin_in.ptr, c.batch, pg.PG_MEM_HOST_PINNED)
            pg.pg_potential(h, pin_out.ptr, c.batch, pg.PG_MEM_HOST_PINNED)
        pg.pg_synchronize(h)

    for _ in range(2):
        b_up(); b_solve(); b_down(); b_all(2)
    t_up, t_sv = med(b_up, 10), med(b_solve, 10)
    t_dn = med(b_down, 10) - t_sv
    t_all = med(b_all, 5) / 6
    pin_in.free(); pin_out.free(); s.close()
    gbs = lambda ms: nbytes / (ms * 1e-3) / 1e9
    line = {
        "metric": "host staging of one 128^3 fp64 array (16.8 MB) through pg_set_density / pg_potential (row a6)",
        "unit": "ms", "n_gpus": 1, "dtype": "f64", "data": "synthetic", "repeats": reps,
        "h2d": {"pinned_ms": h2d_pinned, "pageable_ms": h2d_pageable, "pinned_gbs": gbs(h2d_pinned), "pageable_gbs": gbs(h2d_pageable)},
        "d2h": {"pinned_ms": d2h_pinned, "pageable_ms": d2h_pageable, "pinned_gbs": gbs(d2h_pinned), "pageable_gbs": gbs(d2h_pageable),
                "how": "pg_potential into a host buffer minus the device-resident solve of the same grid"},
        "solve_ms_1024x2048": t_solve, "outputs_equal_and_sane": ok,
        "paper": {"h2d_pinned_ms": 1.0, "h2d_pageable_ms": 3.0, "hardware": "A100 40 GB, PCIe host link", "source": "PAPER.md:119 (section 2.2.2)"},
        "pipeline_config4": {"batch": c.batch, "bytes_each_way": int(np.prod(shape)) * 8, "upload_only_ms": t_up, "solve_only_ms": t_sv,
                             "download_only_ms": t_dn, "sum_ms": t_up + t_sv + t_dn, "pipelined_ms_per_batch": t_all,
                             "note": "pipelined is close to max(upload, download), not to the sum: H2D(b+1), solve(b) and D2H(b-1) overlap"},
        "host": host_placement(0),
    }
    print(json.dumps(line), flush=True)
    return 0


def measure_nested(args):
    """--nested D [--cart N]: the paper's distributed scheme (row NEXT-3): D nested mesh levels of N^3 cells
    (Fig. 8 :306; readings M1-M6).  One process: all levels on one GPU, one CUDA stream each.
    Under torchrun with WORLD_SIZE = D: one level per rank / GPU, the two level-boundary messages by NCCL send / recv.
    A step is one solve of all levels.  Parity gate: the same code path at 32^3 against oracle/nested_oracle.py (the
    oracle's per-level direct sums cost N^6; at the timed size they would take hours)."""
    import torch
    from paper_2409_02294_b200 import binding as pg, build as pg_build, nested
    rank, local_rank, world = replicas.dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if not os.path.exists(pg.LIB_PATH):
        pg_build.build()
    depth, n, box0 = args.nested, (args.cart or 64), 16.0
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if world != depth:
            raise SystemExit(f"bench.py --nested {depth}: one level per rank needs WORLD_SIZE == {depth}, got {world}")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def level_rho(m, level, seed):
        return make_rho3(m, 10 * seed + level)

    # ---- parity gate at 32^3 (rank 0 only runs the oracle; every rank runs its level)
    parity = {"ok": True, "what": "not run"}
    gate_n = 32
    link_kw = dict(link=args.nested_link, token_device=(f"cuda:{local_rank}" if world > 1 else "cpu"))
    gate = nested.NestedPotential(gate_n, box0, depth, device=local_rank, dist=dist, **link_kw)
    g_rho = {l: torch.from_numpy(level_rho(gate_n, l, 1)).cuda() for l in gate.owned}
    g_out = {l: torch.empty_like(g_rho[l]) for l in gate.owned}
    gate.solve(g_rho, g_out); gate.synchronize(); gate.close()
    if rank == 0:
        import oracle
        from oracle import nested_oracle
        ref, _ = nested_oracle.nested_potential(gate_n, box0, [level_rho(gate_n, l, 1) for l in range(depth)])
        got = g_out[0].cpu().numpy()
        l2 = float(np.linalg.norm(got - ref[0]) / np.linalg.norm(ref[0])); mx = float(np.abs(got / ref[0] - 1).max())
        if world == 1:
            for l in range(1, depth):
                g = g_out[l].cpu().numpy()
                l2 = max(l2, float(np.linalg.norm(g - ref[l]) / np.linalg.norm(ref[l]))); mx = max(mx, float(np.abs(g / ref[l] - 1).max()))
        parity = {"rel_l2": l2, "max_rel": mx, "bar": {"rel_l2": REL_L2, "max_rel": MAX_REL}, "ok": bool(l2 <= REL_L2 and mx <= MAX_REL),
                  "what": f"every level this rank owns at {gate_n}^3, depth {depth}, vs oracle/nested_oracle.py (worst level)"}

    # ---- timed region
    npot = nested.NestedPotential(n, box0, depth, device=local_rank, dist=dist, **link_kw)
    R = 2
    d_rho = [{l: torch.from_numpy(level_rho(n, l, r)).cuda() for l in npot.owned} for r in range(R)]
    d_out = [{l: torch.empty_like(d_rho[r][l]) for l in npot.owned} for r in range(R)]
    cur = torch.cuda.current_stream()

    def step(k):
        npot.solve(d_rho[k % R], d_out[k % R])

    def join():
        for l in npot.owned:
            cur.wait_stream(npot.levels[l].stream)

    for k in range(max(3, args.warmup)):
        step(k)
    npot.synchronize()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    rep_ms = []
    n0 = npot.launches()
    for _ in range(REPEATS):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        replicas.barrier(world); torch.cuda.synchronize()
        e0.record(cur)
        for k in range(args.steps):
            step(k)
        join()
        e1.record(cur)
        torch.cuda.synchronize(); replicas.barrier(world)
        rep_ms.append(replicas.max_over_ranks(e0.elapsed_time(e1), world, "cuda"))
    n1 = npot.launches()
    clocks = sampler.stop() if sampler is not None else None
    ms_per_step = float(np.median(rep_ms)) / args.steps
    h3 = pg.pg3_create(n, box0, local_rank, None)
    alg_level = pg.pg3_algorithmic_bytes(h3)
    pg.pg3_destroy(h3)
    n_mean, n_halo = nested.message_counts(n)
    alg = (2 * depth - 1) * alg_level
    peak, peak_src = load_peaks()
    gbs = alg / (ms_per_step * 1e-3) / 1e9 / max(1, world)
    sane = all(bool(torch.isfinite(d_out[0][l]).all() and (d_out[0][l] < 0).all()) for l in npot.owned)
    npot.close()
    line = {
        "metric": "nested-mesh solves/sec (fp64 zero-padded FFT convolution on nested 3-D meshes; row NEXT-3)",
        "value": 1e3 / ms_per_step, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"{depth} nested mesh levels of {n}^3 cells (PAPER.md:267, :269, Fig. 8), box {box0:g} halved per level, "
                               "condensed clump + 6 Gaussian clumps + 1 % noise on every level", "n": n, "depth": depth,
                   "parallelism": ((f"one level per GPU, level-boundary messages "
                                    + ("PUT by the producing kernels into the neighbour's inbox (CUDA IPC peer memory), nccl tokens"
                                       if args.nested_link == "put" else "by NCCL send / recv")) if world > 1
                                   else "all levels on one GPU, one CUDA stream per level"),
                   "exchange_bytes_per_solve": 8 * (depth - 1) * (n_mean + n_halo)},
        "cells_per_s": depth * n**3 * 1e3 / ms_per_step, "gpu_launches": int(round((n1 - n0) / REPEATS)) * world,
        "repeats": {"n": REPEATS, "ms_per_step_median": ms_per_step, "ms_per_step_min": min(rep_ms) / args.steps,
                    "ms_per_step_max": max(rep_ms) / args.steps},
        "parity": parity, "output_sane": sane,
        "roofline": {"bound": "hbm", "kernel": f"whole path ({2 * depth - 1} single-level solves of 7 launches + coupling kernels)",
                     "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None, "peak_source": peak_src,
                     "algorithmic_bytes_per_step": alg, "note": "per GPU"},
        "e2e": {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                "how": "not measured for this row: densities and potentials stay resident (the paper's solver is part of a device-resident code)"},
        "clocks": clocks,
    }
    if world > 1:
        dist.barrier(); dist.destroy_process_group()
    return line, (0 if parity["ok"] else 3)


def run_nested(args):
    line, rc = measure_nested(args)
    if replicas.dist_env()[0] == 0:
        print(json.dumps(line), flush=True)
    if rc:
        sys.stderr.write(f"bench.py: PARITY GATE FAILED: {line['parity']}\n")
    return rc


def measure_cart(args):
    """--cart N: the paper's own per-GPU workload (row NEXT-2): potential of ONE 3-D Cartesian mesh level of N^3 cells
    (N = 64 or 128) by the zero-padded FFT convolution, device resident.  Same protocol as the main
    line: median of REPEATS repeats of the K-step region, buffer rotation beyond L2, parity gate against the 3-D oracle
    on sampled cells, oracle timed on the host cores.  Not the headline metric (BASELINE.json's is the 2-D path)."""
    import torch
    import oracle
    from paper_2409_02294_b200 import binding as pg, build as pg_build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if not os.path.exists(pg.LIB_PATH):
        pg_build.build()
    n, box = args.cart, 10.0
    st = torch.cuda.Stream()
    h = pg.pg3_create(n, box, 0, st.cuda_stream)
    field_bytes = 8 * n**3
    R = int(min(64, max(4, -(-4 * L2_BYTES // (2 * field_bytes)))))
    base = [make_rho3(n, k) for k in range(min(R, 4))]
    d_rho = [torch.from_numpy(np.roll(base[k % len(base)], 7 * (k // len(base)), axis=2)).cuda() for k in range(R)]
    d_phi = [torch.empty_like(d_rho[0]) for _ in range(R)]
    torch.cuda.synchronize()

    def step(k):
        pg.pg3_set_density(h, d_rho[k % R], pg.PG_MEM_DEVICE)
        pg.pg3_potential(h, d_phi[k % R], pg.PG_MEM_DEVICE)

    for k in range(max(3, args.warmup)):
        step(k)
    pg.pg3_synchronize(h)
    sampler = ClockSampler(0)
    rep_ms = []
    n0 = pg.pg3_launch_count(h)
    for _ in range(REPEATS):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(st)
        for k in range(args.steps):
            step(k)
        e1.record(st)
        torch.cuda.synchronize()
        rep_ms.append(e0.elapsed_time(e1))
    n1 = pg.pg3_launch_count(h)
    got = d_phi[0].cpu().numpy()
    t_end = time.perf_counter() + 0.6
    k = 0
    while time.perf_counter() < t_end:
        step(k); k += 1
        if k % 64 == 0:
            pg.pg3_synchronize(h)
    pg.pg3_synchronize(h)
    clocks = sampler.stop()
    ms_per_step = float(np.median(rep_ms)) / args.steps
    # parity gate + oracle timing on a bounded sample of target cells
    rng = np.random.default_rng(n)
    n_t = {32: 4096, 64: 4096, 128: 1024, 256: 128}[n]
    tg = np.unique(np.concatenate([[0, n**3 - 1], rng.integers(0, n**3, n_t)])).astype(np.int64)
    t0 = time.perf_counter()
    ref = oracle.cart_potential_targets(n, box, base[0], tg)
    t_or = time.perf_counter() - t0
    l2 = float(np.linalg.norm(got.reshape(-1)[tg] - ref) / np.linalg.norm(ref))
    mx = float(np.abs(got.reshape(-1)[tg] / ref - 1.0).max())
    ok = bool(l2 <= REL_L2 and mx <= MAX_REL)
    peak, peak_src = load_peaks()
    alg = pg.pg3_algorithmic_bytes(h)
    gbs = alg / (ms_per_step * 1e-3) / 1e9
    # end to end with pinned host buffers
    pin_in, pin_out = pg.PinnedArray((n, n, n)), pg.PinnedArray((n, n, n))
    pin_in.array[...] = base[0]
    for _ in range(3):
        pg.pg3_set_density(h, pin_in.ptr, pg.PG_MEM_HOST_PINNED); pg.pg3_potential(h, pin_out.ptr, pg.PG_MEM_HOST_PINNED)
    pg.pg3_synchronize(h)
    e2e_steps = max(3, min(args.steps, 20))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        pg.pg3_set_density(h, pin_in.ptr, pg.PG_MEM_HOST_PINNED); pg.pg3_potential(h, pin_out.ptr, pg.PG_MEM_HOST_PINNED)
    pg.pg3_synchronize(h)
    t_e2e = (time.perf_counter() - t0) / e2e_steps
    line = {
        "metric": "potential solves/sec (fp64 zero-padded FFT convolution, one 3-D Cartesian mesh level; row NEXT-2)",
        "value": 1e3 / ms_per_step, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"one {n}^3 Cartesian mesh level (PAPER.md:267, :271), box {box:g}, isolated boundary, "
                               "condensed clump + 6 Gaussian clumps + 1 % noise", "n": n,
                   "l2": f"inputs larger than L2: steps rotate over {R} (rho, Phi) buffer pairs"},
        "cells_per_s": n**3 * 1e3 / ms_per_step, "gpu_launches": int(round((n1 - n0) / REPEATS)),
        "repeats": {"n": REPEATS, "ms_per_step_median": ms_per_step, "ms_per_step_min": min(rep_ms) / args.steps,
                    "ms_per_step_max": max(rep_ms) / args.steps},
        "parity": {"rel_l2": l2, "max_rel": mx, "cells": int(len(tg)), "bar": {"rel_l2": REL_L2, "max_rel": MAX_REL}, "ok": ok,
                   "what": "Phi of buffer 0 as the timed region left it vs oracle/cartesian_oracle.c on sampled cells"},
        "roofline": {"bound": "hbm", "kernel": "whole path (7 launches)", "achieved": gbs, "peak": peak, "unit": "GB/s",
                     "frac": gbs / peak, "traffic": None, "peak_source": peak_src, "algorithmic_bytes_per_step": alg},
        "e2e": {"value": 1.0 / t_e2e, "unit": UNIT, "h2d_bytes_per_step": field_bytes, "d2h_bytes_per_step": field_bytes,
                "how": "pg3_set_density + pg3_potential with PG_MEM_HOST_PINNED buffers, wall clock, pg3_synchronize at the end"},
        "clocks": clocks,
        "cpu_baseline": {"value": (len(tg) / n**3) / t_or, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": f"oracle/cartesian_oracle.c (direct sum, gcc -O3 -march=native -fopenmp) on {len(tg)} of {n**3} "
                                   f"target cells ({t_or:.2f} s), extrapolated to the whole mesh by cells"},
        "host": host_placement(0),
    }
    pin_in.free(); pin_out.free()
    pg.pg3_destroy(h)
    return line, (0 if ok else 3)


def run_cart(args):
    line, rc = measure_cart(args)
    print(json.dumps(line), flush=True)
    if rc:
        sys.stderr.write(f"bench.py: PARITY GATE FAILED: {line['parity']}\n")
    return rc


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=5, choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="default line only: skip the `others` block (config 4, --cart 128, --nested 4 --cart 64 at 20 steps)")
    ap.add_argument("--lanes", type=int, default=0, choices=[0, 1, 2, 3, 4], help="solves in flight (0 = 2 for grids of 2^20 cells and more)")
    ap.add_argument("--nested", type=int, default=0, help="D nested 3-D mesh levels of --cart N cells per edge (row NEXT-3; default N = 64); under torchrun with WORLD_SIZE = D one level per GPU")
    ap.add_argument("--batch", type=int, default=0, help="override the config's batch (fields per call); not a BASELINE.json workload")
    ap.add_argument("--nested-link", default="put", choices=["put", "sendrecv"],
                    help="--nested under torchrun: one-sided puts into the neighbours' inboxes (default) or NCCL send / recv of the messages")
    ap.add_argument("--no-fused", action="store_true", help="small grids: force the three-kernel path (PG_OPT_FUSED = 0)")
    ap.add_argument("--accel", action="store_true", help="time the NEXT-4 variant kernels (pg_acceleration, complex-spectrum potential) at --config")
    ap.add_argument("--direct", action="store_true", help="time the direct-summation cross-check kernel (a5) instead")
    ap.add_argument("--cart", type=int, default=0, choices=[0, 32, 64, 128, 256],
                    help="time the 3-D Cartesian mesh path (row NEXT-2) on an N^3 mesh instead")
    ap.add_argument("--staging", action="store_true", help="time row a6 alone: pinned vs pageable staging of a 128^3 array (PAPER.md:119)")
    args = ap.parse_args()
    if args.accel:
        return run_accel(args)
    if args.direct:
        return run_direct(args)
    if args.staging:
        return run_staging(args)
    if args.nested:
        return run_nested(args)
    if args.cart:
        return run_cart(args)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
