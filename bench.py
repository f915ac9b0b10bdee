#!/usr/bin/env python
"""Benchmark of the DG Euler hot path (BASELINE.json: DOF-updates/s, fp64, order 5, 1024^2 cells).

    python bench.py [--gpus N] [--steps K] [--warmup W]           # this repo's CUDA path
    python bench.py --impl reference [--steps K] [--warmup W]     # the CPU oracle, as it stands
    python bench.py --sweep                                       # configs[4]: orders x grids table
    python bench.py --variants                                    # RK(5,4), Cash-Karp, limiter, torque
    torchrun ... bench.py --gpus N --decomp strips                # ONE problem cut into N strips (strong scaling; NEXT-4)

A *step* is one full time step of the hot path on BASELINE configs[3] (planet-disc, 1024^2 cells,
order 5, SSP-RK3): dg_cfl_dt (row a10 of SURVEY.md 8(a); its reduction rides on the previous last
stage) + dg_step = three fused stage kernels covering rows a1..a9, a11, a12.  The metric counts
degrees of freedom as the paper does (nx ny m^2, variables not counted) times the RK
stages executed (a "sub-step").

One JSON line on stdout (rank 0).  Keys beyond the driver's contract:
  roofline      dominant kernel (the fused stage kernel) against the measured HBM copy bandwidth;
                `achieved` = algorithmic bytes per launch / mean CUDA-event duration of the launches
                inside the timed region (events recorded by the library on its own stream).
  fp64          measured DFMA peak of this GPU and the stage kernel's model-flop rate against it.
  cpu_baseline  the oracle (OpenMP build, all host cores) timed on a bounded sample.
  e2e           the same metric through dg_run_host (HOST buffers in, HOST buffers out): every step
                pays the pinned host->device copy of the state, the layout/basis conversion kernels,
                the step, and the device->host copy of the result.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "DOF-updates/sec (fp64, order 5, 1024^2 cells)"
UNIT = "DOF-updates/s"
CFL = 0.2
FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md, used only without MEASURED_PEAKS.json


# ------------------------------------------------------------------------------------------------
DISC_RECIPE = dict(floor=1e-2, taper=0.1, eps_star=0.2)      # workloads.disc defaults


def workload_config(n: int, order: int, replicas: int = 1, literal: bool = False, limiter: int = 0,
                    parallelism: str = "replicas") -> dict:
    """`config` of the JSON line: the workload as it is actually run, including where its disc constants deviate
    from BASELINE.json's text.  The reference arm prints the same dict for the grid it really ran."""
    from paper_1805_01443_b200 import workloads as W
    rec = dict(W.LITERAL_BASELINE_DISC) if literal else dict(DISC_RECIPE)
    state = n * n * 4 * order * order * 8
    dev = ("disc constants as BASELINE.json writes them (floor 1e-6, star softening 0.02; taper 0.05 per SURVEY.md 8(d))"
           if literal else
           f"DEVIATES from BASELINE.json configs[3] (floor 1e-6, star softening 0.02): runs floor {rec['floor']:g}, "
           f"tanh taper {rec['taper']:g}, star softening {rec['eps_star']:g}, because north_star's step list has no limiter "
           f"and the literal constants go negative without one: see DESIGN.md section 3; the literal constants with "
           f"limiter = 1 are timed in the `literal_with_limiter` block of this line")
    return {
        "workload": f"BASELINE configs[3] shape: planet-disc (locally isothermal h=0.05, q=1e-5 planet, frozen bc, "
                    f"wave-killing zone r>2.2, seeded 1e-4 noise), {n}x{n} cells, DG order {order} "
                    f"({order * order} modes x 4 vars per cell), SSP-RK3, CFL {CFL}, dt recomputed every step, "
                    f"limiter {'on' if limiter else 'off'}; {dev}",
        "nx": n, "ny": n, "order": order, "rk": 3, "state_bytes": state,
        "disc_floor": rec["floor"], "disc_taper": rec["taper"], "star_softening": rec["eps_star"], "limiter": limiter,
        "deviates_from_baseline": not literal,
        "l2": "inputs larger than L2: each stage reads >= one %.0f MB state array (L2 is 126 MB); no flush" % (state / 1e6)
        if state > 2 * 126e6 else "state fits L2 and is NOT flushed between steps: L2-assisted number",
        "parallelism": parallelism, "replicas": replicas,
    }


STAGE_IMPL = 0                  # --stage-impl: DG_TUNE_STAGE_IMPL for every context this run creates (0 = library default)


def new_dg(p: dict, **kw):
    """A DG context with this run's --stage-impl applied."""
    from paper_1805_01443_b200 import DG
    from paper_1805_01443_b200.dg import DG_TUNE_STAGE_IMPL
    g = DG(p, **kw)
    if STAGE_IMPL:
        g.set_tuning(DG_TUNE_STAGE_IMPL, STAGE_IMPL)
    return g


def load_peaks() -> tuple[float, str]:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_ read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s; MEASURED_PEAKS.json absent)"


def load_ncu_traffic(order: int, n: int):
    """dram bytes per stage launch from the committed ncu capture (profiles/stage_traffic.csv), or None."""
    path = os.path.join(ROOT, "profiles", "stage_traffic.csv")
    try:
        with open(path) as f:
            rows = [ln.strip().split(";") for ln in f if ln.strip() and not ln.startswith("#")]
        hdr, rows = rows[0], rows[1:]
        idx = {k: i for i, k in enumerate(hdr)}
        vals = [float(r[idx["dram_read_bytes"]]) + float(r[idx["dram_write_bytes"]]) for r in rows
                if int(r[idx["order"]]) == order and int(r[idx["n"]]) == n]
        return sum(vals) / len(vals) if vals else None
    except Exception:
        return None


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting",
               0x10: "sync_boost", 0x100: "display_clock_setting"}

    def __init__(self, index: int, period: float = 0.01):
        self.period, self.samples, self.bits, self.power = period, [], 0, []
        self.ok, self.max_mhz = False, None
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False
        self.th = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    self.bits |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    self.bits |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.ok:
            self.th = threading.Thread(target=self._run, daemon=True)
            self.th.start()

    def stop(self) -> dict:
        if self.th is not None:
            self._stop.set()
            self.th.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0,
                    "note": "NVML unavailable"}
        s = sorted(self.samples)
        reasons = [name for bit, name in self.REASONS.items() if self.bits & bit]
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(s), "power_w_max": max(self.power) if self.power else None}


def visible_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------------------
def stage_bytes_per_launch(p: dict) -> tuple[float, dict]:
    """Algorithmic HBM bytes of one stage launch, averaged over the launches of one step (DESIGN.md
    "Roofline accounting"): arrays of 4 m^2 doubles per cell read or written by each stage --
    stage 1 reads u^n and writes u^(1) (2 arrays; u^(s-1) = u^n), later stages read u^(s-1), u^n and
    write u^(s) (3 arrays; 96 m^2 B per cell-stage, 64 m^2 in stage 1); the last stage
    also reads the initial state in the cells of the wave-killing zone (row a12)."""
    import numpy as np
    nx, ny, m, rk = p["nx"], p["ny"], p["order"], p["rk"]
    state = nx * ny * 4 * m * m * 8
    arrays = 2 + 3 * (rk - 1)
    f_damp = 0.0
    if p["damp_r0"] > 0.0:
        dx, dy = (p["x1"] - p["x0"]) / nx, (p["y1"] - p["y0"]) / ny
        xc = p["x0"] + (np.arange(nx) + 0.5) * dx
        yc = p["y0"] + (np.arange(ny) + 0.5) * dy
        f_damp = float((np.hypot(xc[None, :], yc[:, None]) > p["damp_r0"]).mean())
    per_launch = state * (arrays + f_damp) / rk
    return per_launch, {"state_bytes": state, "arrays_per_step": arrays, "damping_zone_fraction": round(f_damp, 4),
                        "launches_per_step": rk,
                        "per_dof_update": round(per_launch / (nx * ny * m * m), 2)}


def load_exec_counts(order: int, n: int):
    """Executed fp64 thread instructions per stage launch from the committed ncu capture
    (profiles/stage_exec_counts.csv: sm__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum per kernel of
    one step), averaged over the step's launches: (dfma, dmul, dadd) or None."""
    path = os.path.join(ROOT, "profiles", "stage_exec_counts.csv")
    try:
        with open(path) as f:
            rows = [ln.strip().split(";") for ln in f if ln.strip() and not ln.startswith("#")]
        hdr, rows = rows[0], rows[1:]
        idx = {k: i for i, k in enumerate(hdr)}
        sel = [r for r in rows if int(r[idx["order"]]) == order and int(r[idx["n"]]) == n]
        if not sel:
            return None
        return tuple(sum(float(r[idx[k]]) for r in sel) / len(sel) for k in ("dfma", "dmul", "dadd"))
    except Exception:
        return None




def fp64_block(m: int, n: int, stage_ms: float, fp64_peak) -> dict:
    """EXECUTED fp64 work of the stage kernel (instruction counts of the committed ncu capture, FMA = 2 flops) over
    the live CUDA-event time, against the DFMA peak measured on this GPU.  No model flops: the collocation kernel does
    not execute SURVEY.md 8(a)'s modal operation count."""
    ex = load_exec_counts(m, n)
    out = {"peak_tflops": fp64_peak, "peak_source": "dg_probe_fp64_peak: register-resident DFMA loop on this GPU",
           "executed_thread_inst_per_launch": None, "executed_flops_per_cell_stage": None,
           "achieved_executed_tflops": None, "frac_executed": None,
           "source": "profiles/stage_exec_counts.csv (ncu sm__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum)"}
    if ex and stage_ms > 0:
        dfma, dmul, dadd = ex
        flops = 2.0 * dfma + dmul + dadd
        out.update({"executed_thread_inst_per_launch": {"dfma": dfma, "dmul": dmul, "dadd": dadd},
                    "executed_flops_per_cell_stage": flops / (n * n),
                    "achieved_executed_tflops": flops / (stage_ms * 1e-3) / 1e12,
                    "frac_executed": (flops / (stage_ms * 1e-3) / 1e12 / fp64_peak) if fp64_peak else None,
                    "pipe_slots_frac": ((dfma + dmul + dadd) / (stage_ms * 1e-3) / 1e12 / (fp64_peak / 2.0))
                    if fp64_peak else None})
    return out


def literal_block(args, dev, peak) -> dict:
    """BASELINE.json configs[3] with its LITERAL disc constants (floor 1e-6, star softening 0.02) and the paper's
    positivity limiter after every sub-step (limiter = 1): same grid, same order, own timing."""
    import numpy as np
    import torch
    from paper_1805_01443_b200 import DG, workloads as W
    n, m = args.n, args.order
    p, U = W.disc(n, m, planet=True, noise=1e-4, **W.LITERAL_BASELINE_DISC)
    p = dict(p, limiter=1)
    g = new_dg(p)
    g.set_state(torch.from_numpy(U).to(dev))
    del U
    g.limit()
    for _ in range(3):
        g.step(g.cfl_dt(CFL))
    torch.cuda.synchronize()
    steps = max(1, min(args.steps, 50))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g.stage_timing(True)
    l0 = g.launch_count
    e0.record()
    for _ in range(steps):
        g.step(g.cfl_dt(CFL))
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    stage_ms, _ = g.stage_time_ms()
    g.stage_timing(False)
    launches = (g.launch_count - l0) / steps
    S = g.get_state().cpu().numpy()
    ok = bool(np.isfinite(S).all() and (W.evaluate_nodal(p, S)[:, :, 0] > 0).all())
    _, acct = stage_bytes_per_launch(p)
    arrays = step_arrays(p, acct["damping_zone_fraction"])
    gbs = arrays * acct["state_bytes"] / (ms * 1e-3) / 1e9
    g.close()
    return {"config": workload_config(n, m, literal=True, limiter=1), "steps": steps, "ms_per_step": ms,
            "value": W.dof_count(p) * p["rk"] / (ms * 1e-3), "unit": UNIT, "stage_kernel_ms": stage_ms,
            "launches_per_step": launches, "state_valid": ok,
            "roofline": {"bound": "hbm", "kernels": "3 x stage_kernel + 3 x limit_kernel (the last carries wave-killing + CFL)",
                         "algorithmic_arrays_per_step": round(arrays, 3), "achieved": gbs, "peak": peak, "unit": "GB/s",
                         "frac": gbs / peak}}


def run_strips_arm(args) -> dict | None:
    """--decomp strips: ONE problem (the bench workload) cut into N strips of whole cell rows, one rank per GPU
    (strips.DistStrip: NCCL point-to-point halo exchange per sub-step on a side stream, overlapped with the interior
    row segments; all_reduce(MIN) for dt).  Strong scaling.  SURVEY.md 8(e)/(f) NEXT-4; unmeasured on more than one
    GPU in this pool."""
    import socket
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1805_01443_b200 import DG, replicas, strips, workloads as W
    from paper_1805_01443_b200.build import build

    rank, local, size = replicas.world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if not replicas.init("nccl", dev):                       # a single rank still goes through the same code path
        if os.environ.get("TORCHELASTIC_RUN_ID") and os.environ.get("MASTER_PORT"):
            # under torchrun the store is the agent's (a tcp:// rendezvous would wait for a server that never starts)
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
        else:
            s_ = socket.socket()
            s_.bind(("127.0.0.1", 0))
            port = s_.getsockname()[1]
            s_.close()
            dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1, device_id=dev)
    if rank == 0:
        build()
    dist.barrier()
    n, m = args.n, args.order
    p, U = W.disc(n, m, planet=True, noise=1e-4)
    s = strips.DistStrip(DG, p)
    s.set_state(torch.from_numpy(np.ascontiguousarray(U[s.j0:s.j1])).to(dev))
    del U
    for _ in range(max(args.warmup, 3)):
        s.step(s.cfl_dt(CFL))
    torch.cuda.synchronize()
    sampler = ClockSampler(visible_index(local))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.g.launch_count
    dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev0.record()
    for _ in range(args.steps):
        s.step(s.cfl_dt(CFL))
    ev1.record()
    torch.cuda.synchronize()
    dist.barrier()
    clocks = sampler.stop()
    launches = s.g.launch_count - l0
    rows = s.j1 - s.j0
    value, t_ms = replicas.throughput(ev0.elapsed_time(ev1), rows * n * m * m * p["rk"] * args.steps, dev)
    row_bytes = ((n + 31) // 32) * 32 * 4 * m * m * 8
    out = None
    if rank == 0:
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": size, "steps": args.steps,
               "warmup": max(args.warmup, 3), "ms_per_step": t_ms / args.steps, "higher_is_better": True,
               "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
               "config": workload_config(n, m, replicas=1, parallelism="strips"),
               "gpu_launches": int(launches), "clocks": clocks,
               "decomposition": {"strips": size, "rows_per_strip": rows, "exchange": "one row per neighbour per sub-step, "
                                 "NCCL send/recv on a side stream, overlapped with the interior row segments",
                                 "halo_bytes_per_neighbour_per_substep": row_bytes, "substeps_per_step": p["rk"],
                                 "collectives_per_step": "1 all_reduce(MIN) of one double (dt)"},
               "note": "multi-GPU scaling of this mode is unmeasured in this pool (one GPU per run)"}
    dist.barrier()
    dist.destroy_process_group()
    return out


def run_cuda_arm(args) -> dict | None:
    import numpy as np
    import torch
    from paper_1805_01443_b200 import DG, replicas, workloads as W
    from paper_1805_01443_b200.build import build

    rank, local, size = replicas.world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libdg has no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    replicas.init("nccl", dev)
    if rank == 0:
        build()
    replicas.barrier()

    n, m = args.n, args.order
    p, U = W.disc(n, m, planet=True, noise=1e-4)
    dof = W.dof_count(p)
    rk = p["rk"]
    g = new_dg(p)
    Ud = torch.from_numpy(U).to(dev)
    g.set_state(Ud)
    for _ in range(max(args.warmup, 3)):
        g.step(g.cfl_dt(CFL))
    torch.cuda.synchronize()
    fp64_peak = g.probe_fp64_peak() if rank == 0 else None

    sampler = ClockSampler(visible_index(local))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g.stage_timing(True)
    l0 = g.launch_count
    replicas.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev0.record()
    for _ in range(args.steps):
        g.step(g.cfl_dt(CFL))
    ev1.record()
    torch.cuda.synchronize()
    replicas.barrier()
    clocks = sampler.stop()
    launches = g.launch_count - l0
    elapsed_ms = ev0.elapsed_time(ev1)
    stage_ms, n_timed = g.stage_time_ms()
    g.stage_timing(False)
    value, t_ms = replicas.throughput(elapsed_ms, dof * rk * args.steps, dev)
    final = g.get_state().cpu().numpy()
    ok = bool(np.isfinite(final).all() and (W.evaluate_nodal(p, final)[:, :, 0] > 0).all())
    del final

    # ---- end to end through the C-ABI with HOST buffers (H2D + step + D2H inside the timed region) ----
    hin = torch.from_numpy(U).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    ke = max(1, min(args.steps, args.e2e_steps))
    g.run_host(hin, 1, CFL, hout)                      # warm-up
    replicas.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(ke):
        g.run_host(hin, 1, CFL, hout)                  # blocking: returns after the D2H copy
    e2e_s = time.perf_counter() - t0
    replicas.barrier()
    e2e_value, _ = replicas.throughput(e2e_s * 1e3, dof * rk * ke, dev)
    nrun = 20
    t0 = time.perf_counter()
    g.run_host(hin, nrun, CFL, hout)
    e2e_run_value, _ = replicas.throughput((time.perf_counter() - t0) * 1e3, dof * rk * nrun, dev)
    # two contexts in flight, each on its own stream with its own pinned buffers: the H2D copy of one step
    # overlaps the D2H copy of the other (PCIe is full duplex); every step still pays both copies
    e2e_pipe_value, e2e_pipe_ms = None, None
    try:
        ctxs = []
        for _ in range(2):
            st = torch.cuda.Stream(device=dev)
            with torch.cuda.stream(st):
                gi = new_dg(p, stream=st)
            ctxs.append((gi, torch.from_numpy(U).pin_memory(), torch.empty_like(hin).pin_memory()))

        def worker(gi, hi, ho, k):
            torch.cuda.set_device(local)
            for _ in range(k):
                gi.run_host(hi, 1, CFL, ho)

        for gi, hi, ho in ctxs:
            gi.run_host(hi, 1, CFL, ho)                # warm-up
        kp = max(2, ke)
        replicas.barrier()
        torch.cuda.synchronize()
        th = [threading.Thread(target=worker, args=(gi, hi, ho, kp)) for gi, hi, ho in ctxs]
        t0 = time.perf_counter()
        for x in th:
            x.start()
        for x in th:
            x.join()
        pipe_s = time.perf_counter() - t0
        e2e_pipe_value, _ = replicas.throughput(pipe_s * 1e3, dof * rk * kp * 2, dev)
        e2e_pipe_ms = pipe_s * 1e3 / (2 * kp)
        same = bool(torch.equal(ctxs[0][2], hout if ke == 0 else ctxs[1][2]))
        for gi, _, _ in ctxs:
            gi.close()
        del ctxs
    except Exception as exc:                            # pragma: no cover
        e2e_pipe_value, e2e_pipe_ms, same = None, None, False
        sys.stderr.write(f"bench.py: pipelined e2e leg failed: {exc}\n")
    state_bytes = U.nbytes

    if rank != 0:
        replicas.finish()
        return None

    peak, peak_src = load_peaks()
    bpl, acct = stage_bytes_per_launch(p)
    achieved = bpl / (stage_ms * 1e-3) / 1e9 if stage_ms > 0 else 0.0
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": size, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": t_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(n, m, replicas=size),
        "cell_stage_updates_per_s": value / (m * m),
        "state_valid": ok,
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {
            "bound": "hbm", "kernel": ("dg::stage_kernel_fh<M=%d> (fused RK stage, M worker warps + a helper warp: rows a1-a9, a11, a12 + a10 in the last)"
                                       if (m >= 3 and STAGE_IMPL != 1) else
                                       "dg::stage_kernel<M=%d> (fused RK stage: rows a1-a9, a11, a12 + a10 in the last)") % m,
            "stage_impl": STAGE_IMPL,
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": load_ncu_traffic(m, n), "peak_source": peak_src,
            "ms_per_launch": stage_ms, "launches_timed": int(n_timed), "bytes_per_launch": bpl,
            "accounting": acct, "frac_of_nominal_8TBs": achieved / 8000.0,
            "stage_share_of_step": stage_ms * rk / (t_ms / args.steps) if t_ms > 0 else None,
        },
        "fp64": fp64_block(m, n, stage_ms, fp64_peak),
        "e2e": {
            "value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
            "steps": ke, "ms_per_step": e2e_s * 1e3 / ke,
            "call": "dg_run_host(U_in HOST pinned, nsteps=1, cfl, U_out HOST pinned) per step",
            "amortised": {"value": e2e_run_value, "call": f"dg_run_host(..., nsteps={nrun}, ...): one H2D + {nrun} steps + one D2H"},
            "two_in_flight": {"value": e2e_pipe_value, "ms_per_step": e2e_pipe_ms, "results_identical": same,
                              "call": "two contexts on two streams, one host thread each, dg_run_host(nsteps=1) per step: "
                                      "one step's H2D overlaps the other's D2H; every step pays both copies"},
        },
    }
    if size == 1 and not args.no_literal:
        torch.cuda.empty_cache()
        out["literal_with_limiter"] = literal_block(args, dev, peak)
    if size == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(m, budget_s=args.cpu_budget)
    replicas.finish()
    return out


# ------------------------------------------------------------------------------------------------
def _oracle_rate(n: int, order: int, steps: int, warm: int = 0):
    """DOF-updates/s of the oracle (OpenMP build, all cores) on the disc workload at n x n cells."""
    import oracle
    from paper_1805_01443_b200 import workloads as W
    p, U = W.disc(n, order, planet=True, noise=1e-4)
    ref = oracle.RefDG(p, omp=True)
    ref.set_state(U)
    for _ in range(warm):
        ref.step(ref.cfl_dt(CFL))
    t0 = time.perf_counter()
    for _ in range(steps):
        ref.step(ref.cfl_dt(CFL))
    dt = time.perf_counter() - t0
    return W.dof_count(p) * p["rk"] * steps / dt, dt, ref.threads


def cpu_baseline(order: int, budget_s: float = 15.0) -> dict:
    """The oracle as it stands on the host cores, on a bounded sample of the bench workload."""
    import oracle
    oracle.build()
    n = 128
    rate, dt1, threads = _oracle_rate(n, order, 1)                       # one step sizes the sample
    steps = int(max(1, min(40, budget_s / max(dt1, 1e-3))))
    rate, dt, threads = _oracle_rate(n, order, steps)
    return {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"same planet-disc recipe and order {order} at {n}x{n} cells (1/64 of the bench grid), "
                      f"{steps} SSP-RK3 steps with dt recomputed, oracle/ref_dg.cpp -O2 -ffp-contract=off + one "
                      f"OpenMP parallel-for over cell rows, {dt:.1f} s",
            "host_cpus": os.cpu_count()}


def run_reference_arm(args) -> dict | None:
    """--impl reference: the oracle timed on the host cores, same metric and config as the CUDA arm."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return None
    import oracle
    oracle.build()
    m = args.order
    # size the per-step sample so that (steps + warmup) steps end within ~2 minutes
    r0, _, threads = _oracle_rate(32, m, 1, warm=1)
    total = args.steps + args.warmup
    budget = 120.0
    n = 32
    for cand in (64, 128, 256, 512, 1024):
        if cand > args.n:
            break
        if cand * cand * m * m * 3 * total / r0 <= budget:
            n = cand
    rate, dt, threads = _oracle_rate(n, m, args.steps, warm=args.warmup)
    sample = (f"each step = one SSP-RK3 step of the same planet-disc recipe at {n}x{n} cells (order {m})"
              + ("" if n == args.n else f", a bounded sample of the {args.n}x{args.n} workload sized for the time budget")
              + "; oracle/ref_dg.cpp as it stands, OpenMP over cell rows")
    return {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(n, m, replicas=args.gpus),     # the grid the oracle really ran (n <= --n)
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# ------------------------------------------------------------------------------------------------
def run_sweep(args):
    """configs[4]: planet-disc at orders 1..5 x grids; one JSON line per point (1 GPU)."""
    import torch
    from paper_1805_01443_b200 import DG, workloads as W
    from paper_1805_01443_b200.build import build
    build()
    peak, peak_src = load_peaks()
    grids = [int(x) for x in args.sweep_grids.split(",")]
    orders = [int(x) for x in args.sweep_orders.split(",")]
    for n in grids:
        for m in orders:
            p, U = W.disc(n, m, planet=True, noise=1e-4)
            g = new_dg(p)
            g.set_state(torch.from_numpy(U).cuda())
            del U
            for _ in range(5):
                g.step(g.cfl_dt(CFL))
            torch.cuda.synchronize()
            steps = args.sweep_steps
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g.stage_timing(True)
            ev0.record()
            for _ in range(steps):
                g.step(g.cfl_dt(CFL))
            ev1.record()
            torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1)
            stage_ms, _ = g.stage_time_ms()
            g.stage_timing(False)
            bpl, acct = stage_bytes_per_launch(p)
            dof = W.dof_count(p)
            ach = bpl / (stage_ms * 1e-3) / 1e9
            fits_l2 = acct["state_bytes"] * 3 < 126e6
            print(json.dumps({
                "n": n, "order": m, "steps": steps, "dof_updates_per_s": dof * 3 * steps / (ms * 1e-3),
                "cell_stage_updates_per_s": n * n * 3 * steps / (ms * 1e-3), "ms_per_step": ms / steps,
                "stage_ms": stage_ms, "algorithmic_gbs": ach,
                # an HBM fraction only where the three arrays of a stage do not fit the 126 MB L2; below that the
                # state stays L2-resident between stages and the figure is a rate of algorithmic bytes, not of DRAM
                "hbm_frac": None if fits_l2 else ach / peak,
                "algorithmic_gbs_over_hbm_peak": ach / peak,
                "state_mb": acct["state_bytes"] / 1e6, "fits_l2": fits_l2,
            }), flush=True)
            g.close()
            del g
            torch.cuda.empty_cache()


def step_arrays(p: dict, f_damp: float) -> float:
    """Algorithmic state-sized arrays one time step moves (reads + writes), for any scheme / limiter:
    SSP forms: 2 + 3 (rk-1); general schemes: see below; limiter: one more read per sub-step (writes only the
    cells it changes); wave-killing: f_damp."""
    rk = p["rk"]
    lim = bool(p.get("limiter"))
    if rk <= 3:
        arrays, sub = 2 + 3 * (rk - 1), rk
    elif not lim:
        # state form (dg_tables.h): sub-step i reads its input, u^n and the earlier states with a non-zero
        # coefficient, writes one array.  rk 4 (Table 1, low-storage): 2 + 3 + 3 + 3 + 5; rk 5 (Cash-Karp): 2 + 3 + ... + 7
        arrays, sub = (16, 5) if rk == 4 else (27, 6)
    else:
        # with the limiter the sub-steps keep Z_i (their result before the earlier slopes' terms) as well:
        # input, u^n, the earlier Z_j with non-zero coefficient, two arrays written (one in the last sub-step)
        nz = {4: [0, 1, 2, 3, 4], 5: [0, 1, 2, 3, 4, 3]}[rk]
        sub = len(nz)
        arrays = 0
        for i in range(sub):
            arrays += (1 if i == 0 else 2) + nz[i] + (2 if i + 1 < sub else 1)
    if p.get("limiter"):
        arrays += sub
    return arrays + f_damp


def run_variants(args):
    """SURVEY.md 8(f) rows on the bench workload's shape: one JSON line per variant (1 GPU)."""
    import numpy as np
    import torch
    from paper_1805_01443_b200 import DG, workloads as W
    from paper_1805_01443_b200.build import build
    build()
    peak, peak_src = load_peaks()
    n, m = args.n, args.order
    for name, over in (("ssp33 (bench)", {}), ("ssp33 + limiter", {"limiter": 1}),
                       ("rk4: SSP-RK(5,4), paper Table 1 (low-storage form)", {"rk": 4}), ("rk5: Cash-Karp, paper Table 2", {"rk": 5}),
                       ("rk5 + limiter", {"rk": 5, "limiter": 1}), ("ssp33, HLL flux (isothermal)", {"flux": 1})):
        p, U = W.disc(n, m, planet=True, noise=1e-4)
        p.update(over)
        g = new_dg(p)
        g.set_state(torch.from_numpy(U).cuda())
        del U
        for _ in range(3):
            g.step(g.cfl_dt(CFL))
        torch.cuda.synchronize()
        steps = args.sweep_steps
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = g.launch_count
        ev0.record()
        for _ in range(steps):
            g.step(g.cfl_dt(CFL))
        ev1.record()
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1) / steps
        _, acct = stage_bytes_per_launch(dict(p, rk=3))
        arrays = step_arrays(p, acct["damping_zone_fraction"])
        sub = {2: 2, 3: 3, 4: 5, 5: 6}[p["rk"]]
        gbs = arrays * acct["state_bytes"] / (ms * 1e-3) / 1e9
        line = {"variant": name, "n": n, "order": m, "rk": p["rk"], "limiter": p["limiter"], "flux": p["flux"], "sub_steps": sub,
                "steps": steps, "ms_per_step": ms, "ms_per_sub_step": ms / sub,
                "dof_updates_per_s": W.dof_count(p) * sub / (ms * 1e-3),
                "launches_per_step": (g.launch_count - l0) / steps,
                "algorithmic_arrays_per_step": round(arrays, 3), "hbm_gbs": gbs, "hbm_frac": gbs / peak,
                "peak": peak, "peak_source": peak_src}
        if name.startswith("ssp33 (bench)"):
            t0 = g.time
            g.torque(t0)
            torch.cuda.synchronize()
            ev0.record()
            for _ in range(20):
                g.torque(t0)
            ev1.record()
            torch.cuda.synchronize()
            tms = ev0.elapsed_time(ev1) / 20
            tb = acct["state_bytes"] / 4
            line["torque"] = {"ms_per_call": tms, "algorithmic_bytes": tb, "hbm_gbs": tb / (tms * 1e-3) / 1e9,
                              "hbm_frac": tb / (tms * 1e-3) / 1e9 / peak,
                              "note": "dg_torque: density nodes of the whole grid -> 2 kernels + one 24-byte D2H (blocking)"}
        print(json.dumps(line), flush=True)
        g.close()
        del g
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)       # configs[3]: 200 steps
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--n", type=int, default=1024)
    ap.add_argument("--order", type=int, default=5)
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-literal", action="store_true", help="skip the literal_with_limiter block")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "strips"],
                    help="N > 1: independent replicas (default, north_star) or ONE problem cut into N strips along y "
                         "with a halo exchange per sub-step (strips.DistStrip; strong scaling)")
    ap.add_argument("--stage-impl", type=int, default=0, choices=[0, 1, 2],
                    help="DG_TUNE_STAGE_IMPL (include/dg.h): 0 = the library's default stage kernel per order, "
                         "1 = dg::stage_kernel (M worker warps) at every order, 2 = the helper-warp kernel where it exists")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--variants", action="store_true")
    ap.add_argument("--sweep-grids", default="256,512,1024,2048")
    ap.add_argument("--sweep-orders", default="1,2,3,4,5")
    ap.add_argument("--sweep-steps", type=int, default=50)
    args = ap.parse_args()
    global STAGE_IMPL
    STAGE_IMPL = args.stage_impl
    if args.sweep:
        run_sweep(args)
        return
    if args.variants:
        run_variants(args)
        return
    if args.impl == "reference":
        out = run_reference_arm(args)
    elif args.decomp == "strips":
        out = run_strips_arm(args)
    else:
        out = run_cuda_arm(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
