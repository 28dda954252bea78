#!/usr/bin/env python
"""bench.py -- one JSON line for the deposit + fold + apply + return step (BASELINE.json metric).

A "step" is one pass of the whole hot path (pm_deposit, pm_fold_ghosts, pm_apply_limited,
pm_return_to_particles) over the synthetic config-5 workload (512^3 cells, 10^6 particles), all inputs
resident in HBM.  `value` = cell-updates per second (whole job), timed with CUDA events on the stream the
kernels are launched on, barrier + synchronize on both sides, max over ranks.  `e2e` = the same metric through
pm_step_host with pinned HOST buffers (H2D + D2H inside the timed region).  Multi-GPU: the path does not
shard (north_star: one GPU, no collectives), so `--gpus N` runs N independent replicas ("replicas only").

`--impl reference` times the CPU oracle (oracle/pm_oracle.c) as it stands on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "deposit+fold+apply+return step throughput at 512^3, 1e6 particles"
UNIT = "Mcell-updates/s"
ORACLE_SAMPLE_N = 256            # config-5-shaped block the oracle is timed on (same particles per cell)


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            p = [x.strip() for x in ln.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for nm, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(kernel: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed ncu --set full capture,
    profiles/r02_ncu_traffic.csv (made by the command in profiles/r02_ncu_full.md); None if not recorded."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_ncu_traffic.csv")) as f:
            for ln in f.read().splitlines()[1:]:
                k, v = ln.split(",")
                if k == kernel:
                    return float(v)
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------------
def time_oracle(n: int, steps: int, omp: bool = False):
    """The oracle, as it stands, single-threaded: on config 5 itself (n = 512) or on a config-5-shaped n^3 block with the same
    particles per cell (the bounded sample of the default run).  omp=True: the same source compiled with -fopenmp, on all
    host cores."""
    from oracle import pm_oracle as po
    from paper_2509_18261_b200 import inputs
    npart = int(round(1_000_000 * (n / 512.0) ** 3))
    w = inputs.make(5) if n == 512 else inputs.scaled_mixed(n, npart, seed_index=5)
    o = po.Oracle(w.params, w.state, w.sinks, w.sne, keep_abs=False, omp=omp)
    threads = int(po.lib_omp().orc_threads()) if omp else 1
    if omp:
        o.step(w.dt)                      # thread start-up and first touch of the meshes stay outside the timed steps
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(w.dt)
    dt = (time.perf_counter() - t0) / steps
    what = "config 5 itself (512^3, 10^6 particles)" if n == 512 else f"config-5-shaped {n}^3 block, {npart} particles (same particles per cell)"
    how = (f"{threads} OpenMP threads on {os.cpu_count()} host cores (the same source built with -fopenmp: omp atomic deposits, "
           f"parallel particle and cell loops)") if omp else (f"single thread of {os.cpu_count()} host cores (the oracle is a plain "
                                                               f"sequential program)")
    return {"value": n ** 3 / dt / 1e6, "unit": UNIT, "cores": threads, "kind": "oracle, OpenMP build" if omp else "oracle",
            "sample": f"{what}, {steps} step(s), {dt:.2f} s per step, particles/s = {npart / dt:.3e}; {how}",
            "seconds_per_step": dt, "particles_per_s": npart / dt, "steps": steps, "host_cores": os.cpu_count(),
            "workload": "config5_large_512" if n == 512 else f"config5_shape_{n}_{npart} (bounded sample of config5_large_512)"}


def run_reference(args, rank, world):
    """--impl reference: the oracle as it stands on the host cores.  Every step is a bounded sample of the workload (a
    config-5-shaped 256^3 block, ~11 s per step) unless --cpu-baseline-full asks for config 5 itself (~90 s per step); the
    line reports the steps it really ran."""
    if rank != 0:
        return
    n = 512 if args.cpu_baseline_full else ORACLE_SAMPLE_N
    steps = max(1, min(args.steps, 2))
    r = time_oracle(n, steps)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "steps_requested": args.steps, "warmup": 0, "ms_per_step": r["seconds_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": r["workload"], "sample": r["sample"]},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "host_cores")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
def reduce_max(x: float, world: int, device) -> float:
    """Max over ranks of a host scalar (the contract's timing rule); a no-op at world == 1."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def whole_job_value(cells_per_rank: int, steps: int, world: int, total_ms: float) -> float:
    """Mcell-updates/s of the whole job: every rank (replica) updates cells_per_rank cells per step."""
    return world * cells_per_rank * steps / (total_ms * 1e-3) / 1e6


def algorithmic_bytes(N, Nb, nk, nn, t, ts, tn, fk=1.0, fn=1.0, nch=6, Ng=None):
    """Bytes each kernel group must move per step: SURVEY.md 8(d)'s per-cell figures, each touched CELL counted once.
    t, ts, tn = fraction of the owned cells touched by any particle / by a sink / by a supernova; fk, fn = fraction of the
    buffer-mesh tiles that are live in channel group K (accretion) / N (supernovae) -- stale tiles are neither reset nor
    read (pm_tiles.cuh); with every tile live and every cell touched the figures are 8(d)'s dense ones.
    8(d) books "buffer reset + deposit write-back (accumulate in cache, write once)" as ONE row, 8 C_b N_b: it is the
    `zero` entry here (the reset kernels write the live tiles once); the deposit kernels are left with their gather reads
    and the particle records, as in 8(d).  Call it with sector (4-cell) fractions for the bytes DRAM moves at its smallest
    granularity (reported as sector_bytes)."""
    ck, cn = (2, 8) if nch > 6 else (1, 5)                            # Appendix A mode: + count channel, + two error scales
    buf_live = ck * fk + cn * fn                                       # live buffer words per buffer cell
    return {
        "bin": 8.0 * 3 * (nk + nn) + 4.0 * 3 * (nk + nn),            # positions read, keys + perm written and read
        "zero": 8.0 * buf_live * Nb,                                   # a0 + the write-back of a3/a5: each live buffer word written once
        "sinks": 8.0 * 5 * ts * N + 8.0 * 10 * nk,                    # a2: gather 5 fields; particle records
        "sne": 8.0 * 4 * tn * N + 8.0 * 8 * nn,                       # a4: gather 4 fields; particle records
        "fold": 3 * 8.0 * buf_live * (Nb - N if Ng is None else Ng),   # read ghosts, read-modify-write their owned images (Ng: the
                                                                       # ghost cells that can hold anything -- the kernels wrap x at
                                                                       # the source, so only the y and z ghost zones; default: 8(d)'s all)
        "apply": N * (8.0 * buf_live + 96.0 * t + 32.0 * ts),          # live buffer words; 6 + 6 state words and 4 return words where touched
        "return": 8.0 * 4 * ts * N + 8.0 * 12 * nk,
    }


def run_sharded(args, rank, world, local_rank):
    """--sharded: the z-slab decomposition of SURVEY.md 8(f)4.  Rank r holds the planes [n r, n (r + 1)) of a periodic
    n x n x (n world) domain with its own config-5-shaped particle set (weak scaling); a step is the state halo exchange,
    pm_deposit, pm_slab_put (or pm_slab_pack + messages), i.e. the exchange of the buffer's z ghost planes (Eq. 3), pm_fold_ghosts, pm_apply_limited, the
    owner -> ghost copy of the return mesh (R16) and pm_return_to_particles.  With one rank the exchanges are copies onto the
    rank itself and the result is the periodic single-domain step.  Same timing rules as the default arm."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2509_18261_b200 import inputs, pm, sharded

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    n = args.n
    w = inputs.scaled_mixed(n, args.particles, seed_index=5 + rank)
    params = dict(w.params, z_slab=1)
    N, npart = n ** 3, w.sinks.n + w.sne.n
    sk = pm.DeviceSinks.from_host(w.sinks, dev) if w.sinks.n else None
    sn = pm.DeviceSNe.from_host(w.sne, dev) if w.sne.n else None

    def make_ctx(flags):
        c = pm.Context(params, device=str(dev), flags=flags)
        return c, sharded.SlabStep(c, rank, world, peer_put=not args.sharded_messages)

    ctx, stepper = make_ctx(0)
    g = ctx.ghost_width()
    st = pm.DeviceState(*(torch.zeros((n + 2 * g) * n * n, dtype=torch.float64, device=dev) for _ in range(6)))
    for dst, src in zip(st.fields(), w.state.fields()):
        dst.view(n + 2 * g, n, n)[g:g + n].copy_(torch.from_numpy(src))
    d = stepper.d
    xbytes = 2 * (d["buf_send_lo"].numel() + (d["ret_send_lo"].numel() if d["ret_send_lo"] is not None else 0)) * 8 + 6 * 2 * g * n * n * 8
    sampler = ClockSampler(local_rank)
    sampler.start()
    warm = max(args.warmup, 3)
    for _ in range(warm):
        stepper.step(st, sk, sn, w.dt)
    ctx.pm_check()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = ctx.pm_launch_count()
    barrier()
    ev0.record()
    for _ in range(args.steps):
        stepper.step(st, sk, sn, w.dt)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ctx.pm_check()
    launches = ctx.pm_launch_count() - launches0
    total_ms = reduce_max(ev0.elapsed_time(ev1), world, dev)
    ctx.close()
    ctx, stepper = make_ctx(pm.PM_FLAG_TIMING)
    ks = []
    for it in range(5):
        stepper.step(st, sk, sn, w.dt)
        if it >= 2:
            ks.append(ctx.pm_kernel_times())
    kernel_ms = {k: float(np.median([s_[k] for s_ in ks])) for k in pm.KERNEL_GROUPS}
    # e2e: owned planes and particles from pinned host memory every step, result back to the host
    hst = [torch.from_numpy(f).pin_memory() for f in w.state.fields()]
    hsk = {f: torch.from_numpy(getattr(w.sinks, f)).pin_memory() for f in pm.DeviceSinks.IN} if w.sinks.n else None
    hsn = {f: torch.from_numpy(getattr(w.sne, f)).pin_memory() for f in pm.DeviceSNe.IN} if w.sne.n else None
    hout = [torch.empty_like(t) for t in hst]

    def e2e_step():
        for dst, src in zip(st.fields(), hst):
            dst.view(n + 2 * g, n, n)[g:g + n].copy_(src, non_blocking=True)
        if hsk:
            for f in pm.DeviceSinks.IN:
                getattr(sk, f).copy_(hsk[f], non_blocking=True)
        if hsn:
            for f in pm.DeviceSNe.IN:
                getattr(sn, f).copy_(hsn[f], non_blocking=True)
        stepper.step(st, sk, sn, w.dt)
        for dst, src in zip(hout, st.fields()):
            dst.copy_(src.view(n + 2 * g, n, n)[g:g + n], non_blocking=True)
        if hsk:
            for f in ("vx", "vy", "vz", "m"):
                hsk[f].copy_(getattr(sk, f), non_blocking=True)
        torch.cuda.synchronize(dev)

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    for _ in range(e2e_steps):
        e2e_step()
    e2e_s = reduce_max((time.perf_counter() - t0) / e2e_steps, world, dev)
    if rank == 0:
        peak, peak_src = measured_peak()
        Nb = (n + 2 * g) ** 3
        ab = algorithmic_bytes(N, Nb, w.sinks.n, w.sne.n, 1.0, 1.0, 1.0)      # dense 8(d) figures (the fractions are the default arm's business)
        dom = max((k for k in pm.KERNEL_GROUPS if kernel_ms[k] > 0), key=lambda k: kernel_ms[k])
        gbs = ab[dom] / (kernel_ms[dom] * 1e-3) / 1e9
        line = {"metric": METRIC, "value": whole_job_value(N, args.steps, world, total_ms), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": warm, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"config5-shaped {n}^3 slab per rank, z-slab decomposition over {world} rank(s) (--sharded)",
                           "cells_per_rank": N, "particles_per_rank": npart, "multi_gpu": "z slabs, nearest-neighbour exchange of ghost planes: " + ("NCCL point-to-point messages" if args.sharded_messages else "the pack kernel stores into the neighbours' receive slabs through peer memory (CUDA IPC; one host barrier per step)"),
                           "exchange_bytes_per_rank_per_step": xbytes, "l2_policy": "inputs larger than L2"},
                "particles_per_s": world * npart * args.steps / (total_ms * 1e-3), "kernel_ms": kernel_ms, "clocks": clocks,
                "e2e": {"value": world * N / e2e_s / 1e6, "unit": UNIT, "h2d_bytes_per_step": 6 * N * 8 + (7 * w.sinks.n + 8 * w.sne.n) * 8,
                        "d2h_bytes_per_step": 6 * N * 8 + 4 * w.sinks.n * 8, "ms_per_step": e2e_s * 1e3, "steps": e2e_steps,
                        "api": "sharded.SlabStep.step with pinned host buffers copied in and out around it"},
                "gpu_launches": launches,
                "roofline": {"bound": "hbm", "kernel": dom, "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                             "peak_source": peak_src, "traffic": None, "algorithmic_bytes_per_launch": ab[dom],
                             "accounting": "SURVEY.md 8(d) dense figures"},
                "context": "the exchange step of SURVEY 8(f)4; the paper reports ~50% weak-scaling efficiency of its particle update "
                           "to 8192 GPUs (L437); with one rank every exchange is a device copy onto the rank itself"}
        if not args.no_cpu_baseline:
            r = time_oracle(ORACLE_SAMPLE_N, 1)
            line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "host_cores", "workload")}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2509_18261_b200 import inputs, pm

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    n = args.n
    if args.config is not None:             # one of the other BASELINE configs (parity-test workloads; not the headline line)
        w = inputs.make(args.config)
        n = int(w.params["nx"])
    elif n == 512 and args.particles == 1_000_000:
        w = inputs.make(5)
    else:
        w = inputs.scaled_mixed(n, args.particles, seed_index=5)
    N = n ** 3
    Nb = (n + 8) ** 3
    npart = w.sinks.n + w.sne.n
    mode = pm.PM_FLAG_REPRODUCIBLE if args.reproducible else 0
    nch = 9 if args.reproducible else 6
    ctx = pm.Context(w.params, device=str(dev), flags=mode)          # the timed steps run without the per-kernel events
    st = pm.DeviceState.from_host(w.state, dev)
    sk = pm.DeviceSinks.from_host(w.sinks, dev) if w.sinks.n else None
    sn = pm.DeviceSNe.from_host(w.sne, dev) if w.sne.n else None
    stage_names = ("deposit", "fold", "apply", "return")

    def one_step(ev=None):
        if ev: ev[0].record()
        ctx.pm_deposit(st, sk, sn, w.dt)
        if ev: ev[1].record()
        ctx.pm_fold_ghosts()
        if ev: ev[2].record()
        ctx.pm_apply_limited(st)
        if ev: ev[3].record()
        ctx.pm_return_to_particles(sk)
        if ev: ev[4].record()

    sampler = ClockSampler(local_rank)
    sampler.start()                      # nvidia-smi needs ~0.1 s to deliver its first sample: start before the warm-up,
    warm = max(args.warmup, 3)           # so that the (short) timed region is covered; everything until stop() is under load
    for _ in range(warm):
        one_step()
    ctx.pm_check()
    # activity fractions of the buffer the timed steps will see: per cell (SURVEY 8(d)'s unit) and per 32-byte sector (4 cells)
    ctx.pm_deposit(st, sk, sn, w.dt)
    ctx.pm_fold_ghosts()
    n_tiles, live_k, live_n = ctx.debug_tile_counts()           # before the debug view below marks every tile live
    fk, fn = live_k / n_tiles, live_n / n_tiles
    sink_touched = ctx.debug_buffer(0)[1] != 0
    sn_touched = ctx.debug_buffer(1)[1] != 0          # SN d rho > 0 wherever an SN stencil has omega > 0
    touched = sink_touched | sn_touched

    def frac4(m):
        return float(m.reshape(-1, 4).any(dim=1).double().mean())

    t_frac, ts_frac, tn_frac = float(touched.double().mean()), float(sink_touched.double().mean()), float(sn_touched.double().mean())
    t4, ts4, tn4 = frac4(touched), frac4(sink_touched), frac4(sn_touched)
    del touched, sink_touched, sn_touched
    ctx.pm_apply_limited(st)
    ctx.pm_return_to_particles(sk)

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    launches0 = ctx.pm_launch_count()
    barrier()
    for it in range(args.steps):
        one_step(evs[it])
    barrier()
    clocks = sampler.stop()
    launches = ctx.pm_launch_count() - launches0
    ctx.pm_check()
    total_ms = reduce_max(evs[0][0].elapsed_time(evs[-1][4]), world, dev)
    stage_ms = {nm: sum(e[i].elapsed_time(e[i + 1]) for e in evs) / args.steps for i, nm in enumerate(stage_names)}
    ms_per_step = total_ms / args.steps
    value = whole_job_value(N, args.steps, world, total_ms)
    # per-kernel device times: the library's own CUDA events on the launching stream (PM_FLAG_TIMING), three more steps
    ctx.close()
    ctx = pm.Context(w.params, device=str(dev), flags=pm.PM_FLAG_TIMING | mode)
    ksamples = []
    for it in range(5):
        one_step()
        if it >= 2:
            ksamples.append(ctx.pm_kernel_times())
    kernel_ms = {k: float(np.median([s[k] for s in ksamples])) for k in pm.KERNEL_GROUPS}
    # ---- row (f)2b, not part of the step: one sink-creation pass (Sec. 3.1.2) over the same mesh, on copies of the state ----
    creation = None
    if rank == 0 and world == 1 and not args.reproducible:
        ptl = dict(w.params, truelove_J=1.5)
        ctl = pm.Context(ptl, device=str(dev))
        times, found = [], 0
        for rep in range(3):
            cp = pm.DeviceState(*(f.clone() for f in st.fields()))
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            found, _ = ctl.pm_create_sinks(cp, 1 << 20)          # synchronises
            times.append((time.perf_counter() - t0) * 1e3)
            del cp
        ctl.close()
        creation = {"ms": min(times[1:]), "new_sinks": found, "truelove_J": 1.5,
                    "algorithmic_bytes": 8.0 * 3 * N, "timing": "host clock around pm_create_sinks (it synchronises), best of 2 after a warm-up call"}
        creation["achieved_gbs"] = creation["algorithmic_bytes"] / (creation["ms"] * 1e-3) / 1e9
    red_probe = None
    if rank == 0 and world == 1:
        red_probe = {"l2_resident_64MB_5ch": ctx.pm_probe_red_f64(64 << 20, 5),
                     "hbm_footprint_5GB_5ch": ctx.pm_probe_red_f64(5 << 30, 5), "unit": "1e9 fp64 RED lanes/s",
                     "pattern": "rows of 7 consecutive doubles, 5 planes (pm_probe_red_f64)"}

    # ---- the same step through pm_step_graph (one call, replayed from a CUDA graph): what the launch overhead is worth ---------
    graph_leg = None
    if rank == 0 and world == 1:
        torch.cuda.synchronize(dev)                   # the side stream below does not wait for the default stream by itself
        gstream = torch.cuda.Stream(dev)              # a default stream cannot be captured
        with torch.cuda.stream(gstream):
            gctx = pm.Context(w.params, device=str(dev), stream=gstream, flags=mode)
            gst = pm.DeviceState(*(f.clone() for f in st.fields()))
            for i in range(max(warm, 3)):
                gctx.pm_step_graph(gst, sk, sn, w.dt, reuse_args=i > 0)
            gctx.pm_check()
            gsteps = max(args.steps, 10)
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            g0.record()
            for _ in range(gsteps):
                gctx.pm_step_graph(gst, sk, sn, w.dt, reuse_args=True)
            g1.record()
            host_s = time.perf_counter() - t0          # until the last call returns: what the host spends enqueuing
            g1.synchronize()
            graph_leg = {"ms_per_step": g0.elapsed_time(g1) / gsteps, "host_us_per_call": host_s / gsteps * 1e6, "steps": gsteps,
                         "state": gctx.debug_graph_state(),
                         "api": "pm_step_graph: deposit + fold + apply + return captured once, then one cudaGraphLaunch per step; "
                                "CUDA events on the launching stream"}
            gctx.close()
            del gst
        torch.cuda.synchronize(dev)

    # ---- row (f)3, not part of the step: PM gravity (Steps 1, 2, 5; L95, L107) for the same number of particles --------
    gravity = None
    if rank == 0 and world == 1 and not args.reproducible and args.config is None:
        gw = inputs.gravity_workload(n, npart)
        gpos = [torch.from_numpy(a).to(dev) for a in (gw.x, gw.y, gw.z)]
        gvel = [torch.from_numpy(a).to(dev) for a in (gw.vx, gw.vy, gw.vz)]
        gm = torch.from_numpy(gw.m).to(dev)
        gmesh = [torch.from_numpy(a).to(dev) for a in gw.g]
        rho_tot = torch.empty_like(st.rho)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        samples = []
        for rep in range(6):                                         # ctx launches on torch's current stream
            ev[0].record()
            ctx.pm_gravity_deposit(st.rho, gpos[0], gpos[1], gpos[2], gm, rho_tot)
            ev[1].record()
            ctx.pm_gravity_kick(gmesh[0], gmesh[1], gmesh[2], gpos[0], gpos[1], gpos[2], v=gvel, dt=0.5 * gw.dt)
            ev[2].record()
            ctx.pm_drift(gpos[0], gpos[1], gpos[2], gvel[0], gvel[1], gvel[2], gw.dt)
            ev[3].record()
            torch.cuda.synchronize(dev)
            if rep >= 2:
                samples.append([ev[i].elapsed_time(ev[i + 1]) for i in range(3)])
        ctx.pm_check()
        gms = [float(np.median([s_[i] for s_ in samples])) for i in range(3)]
        gbytes = [8.0 * Nb + 24.0 * N + 16.0 * (Nb - N) + 160.0 * npart, 264.0 * npart, 72.0 * npart]
        peak_g, _ = measured_peak()
        gravity = {"particles": npart, "workload": gw.name,
                   "timing": "torch CUDA events on the launching stream, median of 4 after 2 warm-up rounds; meshes (GBs) larger than L2"}
        for name, ms_, b_ in zip(("deposit", "kick", "drift"), gms, gbytes):
            gravity[name] = {"ms": ms_, "algorithmic_bytes": b_, "achieved_gbs": b_ / (ms_ * 1e-3) / 1e9,
                             "frac_of_measured_peak": b_ / (ms_ * 1e-3) / 1e9 / peak_g}
        gravity["particles_per_s_kdk_half"] = npart / (sum(gms) * 1e-3)
        if not args.no_cpu_baseline:       # the gravity oracle as it stands, on a 128^3 block with the same particles per cell
            from oracle import pm_gravity_oracle as go
            ow = inputs.gravity_workload(128, max(npart // 64, 1))
            t0 = time.perf_counter()
            go.gravity_deposit(ow.params, ow.rho_gas, ow.x, ow.y, ow.z, ow.m)
            oa = [go.gravity_interpolate(ow.params, ow.g[c], ow.x, ow.y, ow.z) for c in range(3)]
            ov = [go.kick(v_, a_, 0.5 * ow.dt) for v_, a_ in zip((ow.vx, ow.vy, ow.vz), oa)]
            for c, q in enumerate((ow.x, ow.y, ow.z)):
                go.drift(q, ov[c], ow.dt, 0.0, 128, 1.0)
            osec = time.perf_counter() - t0
            gravity["cpu_baseline"] = {"value": ow.x.size / osec, "unit": "particles/s (one KDK half: deposit + kick + drift)", "cores": 1,
                                       "kind": "oracle", "sample": f"128^3 block, {ow.x.size} particles (same particles per cell), {osec:.3f} s"}
        del gpos, gvel, gm, gmesh, rho_tot

    # ---- e2e through the host-buffer API with pinned host buffers ---------------------------------
    # Every step uploads its own inputs (6 state fields + particles) and downloads its own results inside the timed region.
    # Two host copies of the workload (a host code that double-buffers its mesh) go through the library's two slots in turn
    # (pm_step_host_begin / pm_step_host_end): the upload of one step runs while the step before still downloads.  The
    # one-slot call (pm_step_host: upload, compute, download, wait) is timed as well and reported as `serial_ms_per_step`.
    e2e_steps = max(2, min(max(args.steps, 2), args.e2e_steps))
    hA = inputs.State(*(torch.from_numpy(f).pin_memory() for f in w.state.fields()))
    hB = inputs.State(*(t.clone().pin_memory() for t in hA.fields()))
    class _Host:            # particle arrays in pinned memory too: a copy to or from pageable memory blocks the calling thread
        pass

    def pinned_sinks():
        o = _Host()
        o.n = w.sinks.n
        for f in pm.DeviceSinks.IN:
            setattr(o, f, torch.from_numpy(getattr(w.sinks, f).copy()).pin_memory())
        for f in pm.DeviceSinks.OUT:
            setattr(o, f, torch.zeros(w.sinks.n, dtype=torch.float64).pin_memory())
        return o

    hkA, hkB = pinned_sinks(), pinned_sinks()
    hsn = _Host()
    hsn.n = w.sne.n
    for f in pm.DeviceSNe.IN:
        setattr(hsn, f, torch.from_numpy(getattr(w.sne, f)).pin_memory())
    del st
    torch.cuda.empty_cache()
    ctx.pm_step_host(hA, hkA, hsn, w.dt)      # warm-up (allocates the staging of both slots)
    ctx.pm_step_host_begin(1, hB, hkB, hsn, w.dt)
    ctx.pm_step_host_end(1)
    barrier()
    t0 = time.perf_counter()
    ctx.pm_step_host(hA, hkA, hsn, w.dt)
    torch.cuda.synchronize(dev)
    serial_s = reduce_max(time.perf_counter() - t0, world, dev)
    host = ((hA, hkA), (hB, hkB))
    barrier()
    t0 = time.perf_counter()
    ctx.pm_step_host_begin(0, hA, hkA, hsn, w.dt)
    for i in range(1, e2e_steps):
        ctx.pm_step_host_begin(i % 2, host[i % 2][0], host[i % 2][1], hsn, w.dt)
        ctx.pm_step_host_end((i - 1) % 2)
    ctx.pm_step_host_end((e2e_steps - 1) % 2)
    torch.cuda.synchronize(dev)
    e2e_s = reduce_max((time.perf_counter() - t0) / e2e_steps, world, dev)
    h2d = 6 * N * 8 + 7 * w.sinks.n * 8 + 8 * w.sne.n * 8
    d2h = 6 * N * 8 + 8 * w.sinks.n * 8

    if rank == 0:
        peak, peak_src = measured_peak()
        Ng = n * ((n + 8) ** 2 - n * n)                               # y and z ghost zones of the x-wrapped buffer
        abytes = algorithmic_bytes(N, Nb, w.sinks.n, w.sne.n, t_frac, ts_frac, tn_frac, fk, fn, nch, Ng)
        sbytes = algorithmic_bytes(N, Nb, w.sinks.n, w.sne.n, t4, ts4, tn4, fk, fn, nch, Ng)
        dbytes = algorithmic_bytes(N, Nb, w.sinks.n, w.sne.n, 1.0, 1.0, 1.0, 1.0, 1.0, nch)
        kernels = {}
        for k in pm.KERNEL_GROUPS:
            if kernel_ms[k] > 0:
                gbs = abytes[k] / (kernel_ms[k] * 1e-3) / 1e9
                tr = ncu_traffic(k)
                kernels[k] = {"ms": kernel_ms[k], "algorithmic_bytes": abytes[k], "achieved_gbs": gbs,
                              "frac_of_measured_peak": gbs / peak, "sector_bytes": sbytes[k], "dense_bytes": dbytes[k],
                              "traffic": tr, "traffic_over_algorithmic": (tr / abytes[k]) if tr else None}
        # reset + deposit as the one stage SURVEY 8(d) books them as (a0-a5): write every live buffer word once, gather each
        # touched state cell once, particle records
        a05_ms = sum(kernel_ms[k] for k in ("zero", "sinks", "sne"))
        a05_bytes = sum(abytes[k] for k in ("zero", "sinks", "sne"))
        stage_a0_a5 = {"ms": a05_ms, "algorithmic_bytes": a05_bytes,
                       "achieved_gbs": a05_bytes / (a05_ms * 1e-3) / 1e9 if a05_ms > 0 else None,
                       "frac_of_measured_peak": a05_bytes / (a05_ms * 1e-3) / 1e9 / peak if a05_ms > 0 else None,
                       "kernels": ["k_tiles_mark", "k_tiles_zero", "k_zero_sweep", "k_deposit_sinks_g4", "k_deposit_sne_g3n4"]}
        dom = max(kernels, key=lambda k: kernels[k]["ms"])
        kname = {"sne": "k_deposit_sne_g3n4", "apply": "k_apply_limited", "zero": "k_zero_sweep", "sinks": "k_deposit_sinks_g4",
                 "fold": "k_fold_ghosts", "return": "k_return_sinks_g4", "bin": "k_bin_*"}[dom]
        step_bytes = sum(abytes.values())
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warm, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name + ("+appendixA_reproducible" if args.reproducible else ""), "cells": N, "particles": npart, "sinks": w.sinks.n, "sne": w.sne.n,
                       "multi_gpu": "replicas only" if world > 1 else "single GPU",
                       "l2_policy": "inputs larger than L2 (state 6 fields + 6-channel buffer, GBs >> 126 MB)",
                       "touched_cell_fraction": t_frac, "sink_cell_fraction": ts_frac, "sn_cell_fraction": tn_frac,
                       "touched_sector_fraction": t4, "sink_sector_fraction": ts4, "sn_sector_fraction": tn4,
                       "live_tile_fraction_accretion": fk, "live_tile_fraction_sn": fn},
            "particles_per_s": world * npart * args.steps / (total_ms * 1e-3),
            "stage_ms": stage_ms,
            "kernel_ms": kernel_ms,
            "clocks": clocks,
            "e2e": {"value": world * N / e2e_s / 1e6, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3, "steps": e2e_steps,
                    "serial_ms_per_step": serial_s * 1e3,
                    "api": "pm_step_host_begin / pm_step_host_end, two slots, pinned host buffers: every step uploads its inputs and "
                           "downloads its results; the upload of a step overlaps the download of the step before (two host copies of "
                           "the workload, alternating); serial_ms_per_step is the one-slot pm_step_host"},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": kname, "achieved": kernels[dom]["achieved_gbs"], "peak": peak,
                         "unit": "GB/s", "frac": kernels[dom]["frac_of_measured_peak"], "peak_source": peak_src,
                         "traffic": kernels[dom]["traffic"], "traffic_over_algorithmic": kernels[dom]["traffic_over_algorithmic"],
                         "algorithmic_bytes_per_launch": abytes[dom], "sector_bytes_per_launch": sbytes[dom],
                         "accounting": "SURVEY.md 8(d): each touched CELL once; the reset + write-back of the buffer is the `zero` "
                                       "group's (8(d) row 1), not the deposit kernels'",
                         "launch_ms": kernels[dom]["ms"], "share_of_step": kernels[dom]["ms"] / sum(kernel_ms.values()),
                         "timing": "CUDA events recorded by the library on the launching stream (PM_FLAG_TIMING ctx, after the timed region), median of 3 steps",
                         "frac_of_8tbs_nominal": kernels[dom]["achieved_gbs"] / 8000.0},
            "kernels": kernels,
            "stage_a0_a5": stage_a0_a5,
            "step_roofline": {"algorithmic_bytes_per_step": step_bytes, "sector_bytes_per_step": sum(sbytes.values()),
                              "achieved_gbs": step_bytes / (ms_per_step * 1e-3) / 1e9,
                              "frac_of_measured_peak": step_bytes / (ms_per_step * 1e-3) / 1e9 / peak,
                              "frac_of_8tbs_nominal": step_bytes / (ms_per_step * 1e-3) / 1e9 / 8000.0,
                              "dense_survey_bytes": sum(dbytes.values())},
        }
        if creation:
            line["sink_creation"] = creation
        if graph_leg:
            line["graph_step"] = graph_leg
        if gravity:
            line["gravity"] = gravity
        if red_probe:
            n_red = 5.0 * 183.0 * w.sne.n     # ~183 cells with omega > 0 per SN (SURVEY.md 8 probe), 5 channels
            red_probe["sn_deposit_achieved"] = n_red / (kernel_ms["sne"] * 1e-3) / 1e9 if kernel_ms["sne"] > 0 else None
            line["red_throughput"] = red_probe
        if world == 1 and not args.no_cpu_baseline:
            r = time_oracle(512 if args.cpu_baseline_full else ORACLE_SAMPLE_N, 1)
            line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "host_cores", "workload")}
            # the same source on all host cores (OpenMP); reported beside the single-thread figure
            ro = time_oracle(512 if args.cpu_baseline_full else ORACLE_SAMPLE_N, 2, omp=True)
            line["cpu_baseline_all_cores"] = {k: ro[k] for k in ("value", "unit", "cores", "kind", "sample", "host_cores", "workload")}
        line["context"] = "paper: ~50% weak-scaling efficiency to 8192 MI250X GPUs on Frontier (PAPER.md L9, L437); no throughput published"
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=512, help="cells per side (default: config 5)")
    ap.add_argument("--particles", type=int, default=1_000_000)
    ap.add_argument("--config", type=int, default=None, choices=[1, 2, 3, 4, 5],
                    help="time another BASELINE config instead of config 5 (for the table in DESIGN.md; the headline is config 5)")
    ap.add_argument("--e2e-steps", type=int, default=6)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-baseline-full", action="store_true",
                    help="time the oracle on config 5 itself (512^3, ~90 s per step, ~25 GB of host memory) instead of the bounded 256^3 sample")
    ap.add_argument("--sharded", action="store_true",
                    help="z-slab decomposition (SURVEY 8(f)4): every rank holds one n^3 slab of an n x n x (n world) domain and "
                         "exchanges ghost planes with its z neighbours; default (without the flag): independent replicas")
    ap.add_argument("--sharded-messages", action="store_true",
                    help="with --sharded: send the buffer's ghost planes as NCCL point-to-point messages (pm_slab_pack + send/recv) "
                         "instead of the default, the pack kernel storing them into the neighbours' receive slabs through peer memory "
                         "(pm_slab_put)")
    ap.add_argument("--reproducible", action="store_true",
                    help="Appendix A mode (PM_FLAG_REPRODUCIBLE): 4 more buffer channels + rounding pass; a separate workload variant")
    args = ap.parse_args()
    rank, world, local_rank = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.sharded:
        run_sharded(args, rank, world, local_rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
