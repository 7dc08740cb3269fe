#!/usr/bin/env python
"""bench.py -- the Nekbone CG hot path on B200, one JSON line (contract: task prompt).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config5] [--impl ours|reference]

A "step" is one nk_cg call: cg_init + `niter` CG iterations (ax_e -> gs+mask -> update x,r + rtr,
with pap and the direction update fused into ax_e) over one seeded synthetic RHS, i.e. one pass of
every SURVEY 8(a) row.  Default workload = BASELINE.json configs[4] (E=32768, N=11, 100 iterations),
the largest single-GPU configuration and the one the >= 70 % HBM target is quoted on.

  value        CG fp64 GFLOP/s, model flops (12(N+1)+27 per local point + gs adds) / device time,
               inputs resident in HBM, CUDA events on the launching stream, max over ranks
  e2e          same metric through nk_cg_host: pinned HOST f in, HOST x + history out, inside the timer
  roofline     the dominant kernel (ax_e as it runs inside CG) against the measured HBM copy peak;
               per-launch time from CUDA events recorded between launches IN the timed region
  cpu_baseline the oracle (oracle/, as it stands) on the host cores, on a bounded sample

N > 1 (torchrun): the path is single-GPU; every rank solves an independent replica
of the workload (no data-path collective), "scaling": "weak".
`--impl reference` times the oracle (this tier's reference arm) on rank 0 only.
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

import numpy as np

METRIC = "nekbone_cg_fp64_gflops"
UNIT = "GFLOP/s"
HBM_NOMINAL_GBS = 8000.0          # BASELINE.json: "fraction of ~8 TB/s"
HBM_FALLBACK_GBS = 6650.0         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent


# ---- model -----------------------------------------------------------
def flops_per_point_iter(N: int, gs_adds_per_pt: float) -> float:
    """ax_e 12(N+1)+15, pap 3, update+rtr 7, p update 2 (= 12(N+1)+27) + gs adds."""
    return 12.0 * (N + 1) + 27.0 + gs_adds_per_pt


def gs_bytes(sizes: dict) -> float:
    """20 B per listed local copy (8 read + 8 write + 4 index) + 4 B per CSR row."""
    return 20.0 * sizes["n_listed"] + 4.0 * sizes["n_rows"]


def gs_gather_bytes(L: int, sizes: dict) -> float:
    """gs folded into the residual update: a dense 4-byte gather code per local point, and per listed local copy
    one 8-byte gather (the partner of a face point; the copies of an edge or corner node are read once per copy
    too); nothing is written back."""
    return 4.0 * L + 8.0 * sizes["n_listed"]


def iter_model_bytes(L: int, sizes: dict) -> float:
    """Canonical unfused per-iteration model: 168 B/pt + gs."""
    return 168.0 * L + gs_bytes(sizes)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback"


# ---- clocks during the timed region ---------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.thread, self.index = [], None, None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for ts, line in self.rows:
            if ts < t0 or ts > t1 + 0.1:
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(self.NAMES, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:   # region shorter than one sample: use whatever was seen
            for ts, line in self.rows[-3:]:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
                except (ValueError, IndexError):
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(smax)) if smax else None,
                "power_w_max": float(max(power)) if power else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- the oracle, timed (cpu_baseline and --impl reference) ------------------------------------------
def cpu_model_name() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


class OracleRun:
    """The oracle (test infrastructure, timed as it stands) set up on the WORKLOAD'S OWN mesh: a step of the
    CPU arm is k CG iterations of the real problem (cg_init + k iterations), not a smaller stand-in."""

    def __init__(self, workload: str, mesh=None, f=None):
        from oracle.nko import Oracle, num_threads
        from workloads import CONFIGS, config_mesh, rhs_unique
        cfg = CONFIGS[workload]
        self.workload, self.cfg = workload, cfg
        self.mesh = config_mesh(workload) if mesh is None else mesh
        self.f = rhs_unique(self.mesh, cfg["seed"]) if f is None else f
        t = time.perf_counter()
        self.orc = Oracle.from_mesh(self.mesh)
        self.setup_s = time.perf_counter() - t
        self.cores = int(num_threads())
        s = self.orc.sizes()
        self.gs_adds = float(self.mesh.L - s["n_unique"]) / self.mesh.L
        self.fpp = flops_per_point_iter(cfg["N"], self.gs_adds)

    def time_iters(self, k: int) -> float:
        t = time.perf_counter()
        self.orc.cg(self.f, k)
        return time.perf_counter() - t

    def iters_for(self, budget_s: float) -> int:
        """k >= 3 iterations per step (never more than the workload's own count) that fit the budget."""
        self.time_iters(1)                                # first call: thread pool, page faults
        t1, t4 = self.time_iters(1), self.time_iters(4)   # a call has a fixed part (cg_init, allocations)
        per = max((t4 - t1) / 3.0, 1e-7)
        return int(max(3, min(self.cfg["niter"], (budget_s - max(t1 - per, 0.0)) / per)))

    def gflops(self, k: int, seconds: float) -> float:
        return self.fpp * self.mesh.L * k / seconds / 1e9

    def describe(self, k: int) -> str:
        m = self.mesh
        full = " (the whole solve)" if k == self.cfg["niter"] else f" of the solve's {self.cfg['niter']}"
        return (f"oracle nko_cg on the workload's own mesh (E={m.E}, N={m.N}, L={m.L}): cg_init + {k} CG iterations"
                f"{full}")

    def best_of(self, fn, reps=5, warm=1):
        for _ in range(warm):
            fn()
        ts = []
        for _ in range(reps):
            t = time.perf_counter()
            fn()
            ts.append(time.perf_counter() - t)
        return min(ts)

    def kernels(self) -> dict:
        """ax_e and gs(+mask), best of 5 wall-clock applications."""
        from workloads import field_local
        m = self.mesh
        u = field_local(m, 1004)
        t_ax = self.best_of(lambda: self.orc.ax_e(u))
        t_gs = self.best_of(lambda: self.orc.mask(self.orc.gs(u)))
        fl = (12.0 * (m.N + 1) + 15.0) * m.L
        return {"ax_e": {"ms": 1e3 * t_ax, "gflops": fl / t_ax / 1e9, "gbs_model": 64.0 * m.L / t_ax / 1e9},
                "gs_mask": {"ms": 1e3 * t_gs}}


def cpu_baseline(workload: str, mesh=None, f=None, budget_s: float = 12.0) -> dict:
    from oracle import nko
    s = OracleRun(workload, mesh, f)
    k = s.iters_for(budget_s)
    sec = s.time_iters(k)
    out = {"value": s.gflops(k, sec), "unit": UNIT, "cores": s.cores, "kind": "oracle",
           "sample": s.describe(k), "seconds": sec, "cpu": cpu_model_name(), "oracle_setup_s": s.setup_s,
           "note": "plain C99 loops + OpenMP parallel for (oracle/nko.c as it stands, untuned)"}
    out["kernels"] = s.kernels()
    # one-thread figure, on the same mesh, at most ~10 s
    nko.set_num_threads(1)
    try:
        k1 = max(1, min(k, int(10.0 / max(sec / k * s.cores, 1e-9))))     # assumes perfect scaling: an upper bound on its time
        t1 = s.time_iters(k1)
        out["one_thread"] = {"value": s.gflops(k1, t1), "unit": UNIT, "iterations": k1, "seconds": t1}
    finally:
        nko.set_num_threads(s.cores)
    return out


def run_reference(args) -> dict:
    """This tier's reference arm: the oracle on the host cores, on the workload's own mesh; a step is cg_init +
    k CG iterations, k sized so that the whole --steps/--warmup run ends within a few minutes."""
    from workloads import CONFIGS
    s = OracleRun(args.workload)
    total_budget = 150.0                                  # whole run within a few minutes
    k = s.iters_for(total_budget / max(1, args.steps + args.warmup))
    for _ in range(args.warmup):
        s.time_iters(k)
    t = 0.0
    for _ in range(args.steps):
        t += s.time_iters(k)
    val = s.gflops(k * args.steps, t)
    cfg = CONFIGS[args.workload]
    conf = workload_config(args.workload, cfg, args.gpus)
    conf["step"] = f"cg_init + {k} CG iterations of the workload's mesh (of its {cfg['niter']}; GFLOP/s is per iteration work)"
    conf["iterations_per_step"] = k
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "gpu_launches": 0, "config": conf,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": s.cores, "kind": "oracle",
                             "sample": s.describe(k) + " per step", "cpu": cpu_model_name(),
                             "oracle_setup_s": s.setup_s},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def workload_config(name: str, cfg: dict, n_gpus: int) -> dict:
    nx, ny, nz = cfg["brick"]
    n = cfg["N"] + 1
    return {"workload": f"{name}: E={nx * ny * nz} ({nx}x{ny}x{nz} brick), N={cfg['N']}, "
                        f"amplitude {cfg['amplitude']}, boundary mask, f uniform[-1,1) seed {cfg['seed']}, "
                        f"CG {cfg['niter']} iterations",
            "E": nx * ny * nz, "N": cfg["N"], "n_local": nx * ny * nz * n ** 3, "niter": cfg["niter"],
            "step": "one nk_cg call (cg_init + niter iterations)",
            "parallelism": "single GPU" if n_gpus == 1 else f"{n_gpus} independent replicas (no collective)",
            "l2": "inputs larger than L2" if nx * ny * nz * n ** 3 * 8 * 11 > 2 * 126e6 else "L2-resident: L2 flushed between steps"}


# ---- rank plumbing (no data-path collective: the path is single-GPU, N ranks = N replicas) ------------
def replica_seed(seed: int, rank: int) -> int:
    """Replica `rank` solves the same mesh with its own RHS."""
    return int(seed) + 7919 * int(rank)


def max_over_ranks(dist, values, device):
    """Element-wise MAX over ranks of a short list of timings (ms); identity without a process group."""
    import torch
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(flops_per_step_per_rank: float, steps: int, world: int, ms_max: float) -> float:
    """Aggregate GFLOP/s over all replicas: every rank did `steps` steps within the slowest rank's time."""
    return world * flops_per_step_per_rank * steps / (ms_max * 1e-3) / 1e9


# ---- our arm -----------------------------------------------------------------------------------------
def run_ours(args) -> dict | None:
    import torch
    from paper_2606_12650_b200 import Nekbone          # raises if libnk.so is missing: no fallback
    from workloads import CONFIGS, config_mesh, rhs_unique

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = CONFIGS[args.workload]
    niter, N = cfg["niter"], cfg["N"]
    mesh = config_mesh(args.workload)
    f_np = rhs_unique(mesh, replica_seed(cfg["seed"], rank))
    t0 = time.perf_counter()
    nk = Nekbone.from_mesh(mesh)
    setup_s = time.perf_counter() - t0
    setup_info = nk.setup_info()                           # who built the gs plan, and the library's own clock
    for k, v in (("fuse_pap", args.fuse_pap), ("fuse_p", args.fuse_p), ("fuse_gs", args.fuse_gs), ("graph", args.graph),
                 ("pdl", args.pdl), ("coop", args.coop), ("defer_x", args.defer_x)):
        if v is not None:                                  # None: the library's default
            nk.set_option(k, v)
    sizes = {**nk.sizes(), **nk.gs_sizes()}
    L = mesh.L
    gs_adds = float(L - sizes["n_unique"]) / L
    flops_step = flops_per_point_iter(N, gs_adds) * L * niter
    stream = torch.cuda.current_stream()

    f = torch.from_numpy(f_np).cuda()
    x = nk.empty()
    hist = torch.empty(niter + 1, dtype=torch.float64, device="cuda")
    small = L * 8 * 11 <= 2 * 126e6                                # working set not >> L2: flush between steps
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if small else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if flush is not None:
            flush.fill_(1)
        nk.cg(f, niter, x=x, res_hist=hist)

    # ---- device-resident timed region: the DEFAULT path (no per-launch events: programmatic dependent
    # launches / graph replay exactly as a caller of nk_cg gets them) ---------------------------------------
    for _ in range(args.warmup):
        step()
    barrier()
    nk.set_option("profile", 0)
    solve_path = nk.solve_path()
    launches0 = nk.launch_count()
    clocks = ClockSampler(local)
    clocks.start()
    time.sleep(0.25)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps)]
    barrier()
    w0 = time.time()
    for s in range(args.steps):
        if flush is not None:
            flush.fill_(1)
        ev[2 * s].record(stream)
        nk.cg(f, niter, x=x, res_hist=hist)
        ev[2 * s + 1].record(stream)
    barrier()
    w1 = time.time()
    ms = sum(ev[2 * s].elapsed_time(ev[2 * s + 1]) for s in range(args.steps))
    launches = nk.launch_count() - launches0
    res_final = float(hist[-1])
    # ---- per-kernel breakdown: extra steps with a CUDA event between consecutive launches ("profile": plain
    # launches, no overlap between a kernel's tail and its successor's prologue), clocks still being sampled
    nk.set_option("profile", 1)
    nk.kernel_times()
    prof_steps = max(1, min(3, args.steps))
    for _ in range(prof_steps):
        step()
    ktimes = nk.kernel_times()
    nk.set_option("profile", 0)
    barrier()
    clk = clocks.stop(w0, time.time())
    ktimes_from = (f"{prof_steps} extra step(s) right after the timed region with a CUDA event between consecutive "
                   "launches (option profile=1: plain launches); the timed steps themselves run the default path")
    ms_prof_step = sum(t for t, n in ktimes.values()) / prof_steps

    # ---- end to end through the C-ABI with pinned HOST buffers, copies inside the timer ----------------------------
    # every step copies its right-hand side in and its solution + history out.  One call per step (nk_cg_host:
    # copy, solve, copy, synchronise) is always timed; where no L2 flush between steps is needed (inputs larger than
    # L2) the same steps also run as ONE nk_cg_host_batch call, which overlaps the copies of step j+1 / j-1 with
    # solve j -- the headline e2e number then is the pipelined one, and the serial one is reported beside it.
    f_pin = torch.from_numpy(f_np).pin_memory()
    x_pin = torch.empty(L, dtype=torch.float64).pin_memory()
    h_pin = torch.empty(niter + 1, dtype=torch.float64).pin_memory()
    nk.cg_host(f_pin.numpy(), niter, x_pin.numpy(), h_pin.numpy())           # warm-up
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        if flush is not None:
            flush.fill_(1)
        nk.cg_host(f_pin.numpy(), niter, x_pin.numpy(), h_pin.numpy())
    e1.record(stream)
    barrier()
    ms_e2e_serial = e0.elapsed_time(e1)
    ms_e2e, e2e_mode = ms_e2e_serial, "one nk_cg_host call per step"
    if flush is None:
        x2_pin = torch.empty(L, dtype=torch.float64).pin_memory()
        h2_pin = torch.empty(niter + 1, dtype=torch.float64).pin_memory()
        fs = [f_pin.numpy()] * args.steps
        xs = [(x_pin, x2_pin)[j & 1].numpy() for j in range(args.steps)]
        hs = [(h_pin, h2_pin)[j & 1].numpy() for j in range(args.steps)]
        nk.cg_host_batch(fs[:2], niter, xs[:2], hs[:2])                       # warm-up (streams, events)
        barrier()
        e0.record(stream)
        nk.cg_host_batch(fs, niter, xs, hs)
        e1.record(stream)
        barrier()
        ms_e2e, e2e_mode = e0.elapsed_time(e1), "one nk_cg_host_batch call for all steps (copies overlap the solves)"
        assert args.steps < 2 or np.array_equal(x_pin.numpy(), x2_pin.numpy())

    ms, ms_e2e, ms_e2e_serial = max_over_ranks(dist, [ms, ms_e2e, ms_e2e_serial], "cuda")
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return None

    peak, peak_kind = measured_peaks()
    value = whole_job_value(flops_step, args.steps, world, ms)
    e2e = whole_job_value(flops_step, args.steps, world, ms_e2e)
    opts = {k: nk.get_option(k) for k in ("fuse_pap", "fuse_p", "fuse_gs", "graph", "pdl", "coop", "defer_x")}
    fused_p = opts["fuse_p"] != 0
    fused_gs = bool(opts["fuse_pap"]) and (opts["fuse_gs"] == 1 or (opts["fuse_gs"] == 2 and L >= (1 << 20)))
    # "defer_x": two iterations share one pass over x (24 + 48 B/pt per pair instead of 2 x 40; an odd last one is plain)
    px_bytes = (72.0 * (niter // 2) + 40.0 * (niter % 2)) / max(niter, 1) if opts["defer_x"] else 40.0
    xr_fused_p = (80.0 * (niter // 2) + 48.0 * (niter % 2)) / max(niter, 1) if opts["defer_x"] else 48.0
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(args.workload, cfg, world),
           "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 8 * L,
                   "d2h_bytes_per_step": 8 * (L + niter + 1), "ms_per_step": ms_e2e / args.steps, "mode": e2e_mode,
                   "serial_value": whole_job_value(flops_step, args.steps, world, ms_e2e_serial),
                   "serial_ms_per_step": ms_e2e_serial / args.steps},
           "gpu_launches": int(launches), "clocks": clk,
           "options": {**opts, "solve_path": solve_path, "pdl_effective": nk.pdl_effective(),
                       "fuse_p_effective": int(fused_p), "fuse_gs_effective": int(fused_gs),
                       "profile_in_timed_region": False},
           "setup_s": setup_s, "setup": setup_info, "final_residual": res_final}

    # ---- iteration-level and kernel-level bandwidth ---------------------------------------------------
    # real bytes per point of each kernel class as launched: ax_e u 8 + G 48 + w 8 (+ r 8 read and
    # p 8 written when the direction update is folded in); gs by its plan; the vector kernels by what they touch
    gsb = gs_bytes(sizes) / L
    kb = {"ax_e": 64.0 + (16.0 if fused_p else 0.0), "gs": gsb, "dot": 17.0,
          # the fused gs update takes its weights from the gather code: no 1-byte multiplicity code there
          # ... and with "fuse_p" + "defer_x" a pair costs 24 + 56 B/pt instead of 2 x 48 (x read and written once)
          "update_xr": ((xr_fused_p if fused_p else 24.0) + gs_gather_bytes(L, sizes) / L) if fused_gs
                       else (49.0 if fused_p else 25.0),
          "update_p": 24.0 if fused_p else px_bytes, "cg_init": 33.0}
    it_bytes = iter_model_bytes(L, sizes)
    it_gbs = it_bytes * niter * args.steps / (ms * 1e-3) / 1e9
    real_bpp = sum(kb[k] * n for k, (t, n) in ktimes.items() if k != "cg_init") / (prof_steps * niter)
    real_gbs = real_bpp * L * niter * args.steps / (ms * 1e-3) / 1e9
    out["iteration"] = {"ms_per_iteration": ms / args.steps / niter,
                        "model_bytes_per_point": it_bytes / L, "gbs_model": it_gbs,
                        "frac_model_bytes_of_copy_peak": it_gbs / peak,
                        "frac_model_bytes_of_nominal_8TBs": it_gbs / HBM_NOMINAL_GBS,
                        "model": "canonical UNFUSED iteration of SURVEY 8(d): 168 B/pt + gs; fusion removes real traffic, "
                                 "so this rate can exceed the copy peak -- the real-bytes figures are the physical ones",
                        "real_bytes_per_point": real_bpp, "gbs_real": real_gbs,
                        "frac_real_of_measured_copy": real_gbs / peak,
                        "frac_real_of_nominal_8TBs": real_gbs / HBM_NOMINAL_GBS,
                        "gdofs_paper_eq1": mesh.E * N ** 3 * niter * args.steps / (ms * 1e-3) / 1e9}
    ax_ms, ax_n = ktimes["ax_e"]
    if ax_n > 0:
        bpp = kb["ax_e"]
        avg = ax_ms / ax_n
        ach = bpp * L / (avg * 1e-3) / 1e9
        traffic, traffic_source = args.traffic, "--traffic argument"
        if traffic is None:
            try:
                with open(os.path.join(ROOT, "profiles", "traffic.json.txt")) as fh:
                    rec = json.load(fh)[args.workload if fused_p else args.workload + "_ax_e_alone"]
                traffic = float(rec["dram_bytes_per_launch"])
                traffic_source = ("constant from the committed ncu --set full capture " + rec.get("source", "under profiles/")
                                  + " (dram__bytes_read.sum + dram__bytes_write.sum per launch); NOT measured in this run")
            except Exception:
                traffic, traffic_source = None, None
        out["roofline"] = {"kernel": "ax_tma_kernel (ax_e" + (" + fused p=r+beta*p" if fused_p else "")
                                     + (" + fused pap" if opts["fuse_pap"] else "") + ")",
                           "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                           "peak_kind": peak_kind + " copy peak (burst)", "frac_of_nominal_8TBs": ach / HBM_NOMINAL_GBS,
                           "bytes_per_point": bpp, "avg_launch_us": 1e3 * avg, "launches_timed": ax_n,
                           "traffic": traffic, "traffic_source": traffic_source,
                           "algorithmic_bytes_per_launch": bpp * L,
                           "share_of_step": ax_ms / prof_steps / ms_prof_step,
                           "timed_by": ktimes_from}
        out["kernels"] = {k: {"avg_us": 1e3 * t / n, "launches_per_step": n // prof_steps,
                              "share_of_step": t / prof_steps / ms_prof_step, "real_bytes_per_point": kb[k],
                              "gbs_real": kb[k] * L / (t / n * 1e-3) / 1e9}
                          for k, (t, n) in ktimes.items() if n > 0}
        out["kernels"]["_profiled_step_ms"] = ms_prof_step
        # secondary roofline: the fp64 pipe.  Executed flops of ax_e per point with the even-odd
        # transforms: 6 line transforms of n/2 + 2 fp64 instructions per point (n^2/2 DFMA + 2n DADD per line) =
        # 6(n+1) flops, the 3x3 G 15, the fused pap 6, the final sum 2 -- against a DFMA-only microbenchmark
        n = N + 1
        from paper_2606_12650_b200.binding import fp64_peak
        pk = fp64_peak()
        ex_flops = (6.0 * (n + 1) + 15.0 + (6.0 if opts["fuse_pap"] else 0.0) + 2.0) * L
        ex_instr = (3.0 * n + 12.0 + 9.0 + (4.0 if opts["fuse_pap"] else 0.0) + 2.0) * L
        out["fp64"] = {"peak_tflops_measured": pk["tflops"], "how": "nk_fp64_peak: DFMA-only microbenchmark, 2 flops per DFMA, "
                       "full occupancy, best of 5", "dfma_per_clk_per_sm_at_max_clock": pk["dfma_per_clk_per_sm_at_max_clock"],
                       "ax_e_model_tflops": (12.0 * n + 15.0) * L / (avg * 1e-3) / 1e12,
                       "ax_e_executed_tflops": ex_flops / (avg * 1e-3) / 1e12,
                       "ax_e_fp64_instr_per_s_over_peak_dfma_per_s": ex_instr / (avg * 1e-3) / (pk["tflops"] * 1e12 / 2.0)}
    else:
        out["roofline"] = None
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, mesh, f_np)
    return out


# ---- our arm, sharded: ONE mesh over all ranks ------------------------------------------
def run_sharded(args) -> dict | None:
    """`--sharded`: the workload's mesh is partitioned by elements over the ranks (paper_2606_12650_b200.dist /
    nk_dist_cg: one neighbour-wise halo exchange and two all-gathers of a double per iteration over NCCL), so total
    work is fixed: "strong" scaling.  The default without the flag stays N independent replicas.  Needs a process group
    also at N = 1 (then it measures what the split-phase path costs against the fused nk_cg)."""
    import torch
    import torch.distributed as dist
    from paper_2606_12650_b200.dist import DistNekbone, TorchComm
    from workloads import CONFIGS, config_mesh, rhs_unique

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world == 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", str(29400 + os.getpid() % 500))
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    cfg = CONFIGS[args.workload]
    niter, N = cfg["niter"], cfg["N"]
    mesh = config_mesh(args.workload)
    f_np = rhs_unique(mesh, cfg["seed"])                                  # one RHS for the whole mesh
    d = DistNekbone.from_mesh(mesh, TorchComm())
    L = mesh.L
    U = int(np.unique(mesh.glo_num).size)
    flops_step = flops_per_point_iter(N, float(L - U) / L) * L * niter    # of the WHOLE mesh
    stream = torch.cuda.current_stream()
    f_loc = d.local(f_np)
    f = torch.from_numpy(f_loc).cuda()
    x = d.empty()
    hist = torch.empty(niter + 1, dtype=torch.float64, device="cuda")
    small = d.L * 8 * 11 <= 2 * 126e6
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if small else None

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    def timed(fn):
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps)]
        barrier()
        for s in range(args.steps):
            if flush is not None:
                flush.fill_(1)
            e[2 * s].record(stream)
            fn()
            e[2 * s + 1].record(stream)
        barrier()
        return sum(e[2 * s].elapsed_time(e[2 * s + 1]) for s in range(args.steps))

    for _ in range(args.warmup):
        d.cg(f, niter, x=x, res_hist=hist)
    launches0 = d.nk.launch_count()
    clocks = ClockSampler(local)
    clocks.start()
    time.sleep(0.25)
    w0 = time.time()
    ms = timed(lambda: d.cg(f, niter, x=x, res_hist=hist))
    w1 = time.time()
    clk = clocks.stop(w0, w1)
    launches = d.nk.launch_count() - launches0
    f_pin = torch.from_numpy(f_loc).pin_memory()
    x_pin = torch.empty(d.L, dtype=torch.float64).pin_memory()
    h_pin = torch.empty(niter + 1, dtype=torch.float64).pin_memory()

    def e2e_step():
        f.copy_(f_pin, non_blocking=True)
        d.cg(f, niter, x=x, res_hist=hist)
        x_pin.copy_(x, non_blocking=True)
        h_pin.copy_(hist, non_blocking=True)
        stream.synchronize()

    e2e_step()
    ms_e2e = timed(e2e_step)
    ms, ms_e2e = max_over_ranks(dist, [ms, ms_e2e], "cuda")
    res_final = float(hist[-1])
    n_nbr, n_xch, n_if_el = d.n_neighbors, d.n_exchange, d.n_interface_elements
    dist.barrier()
    dist.destroy_process_group()
    if rank != 0:
        return None
    out = {"metric": METRIC, "value": flops_step * args.steps / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
           "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {**workload_config(args.workload, cfg, world),
                      "parallelism": f"element partition over {world} rank(s): per iteration one neighbour-wise halo exchange "
                                     f"(rank 0: {n_nbr} neighbours, {n_xch} doubles each way, overlapped with ax_e on the "
                                     f"{d.nk.E - n_if_el} interior elements) + 2 all-gathers of one double (NCCL)"},
           "e2e": {"value": flops_step * args.steps / (ms_e2e * 1e-3) / 1e9, "unit": UNIT,
                   "h2d_bytes_per_step": 8 * d.L, "d2h_bytes_per_step": 8 * (d.L + niter + 1),
                   "ms_per_step": ms_e2e / args.steps},
           "gpu_launches": int(launches), "clocks": clk, "final_residual": res_final,
           "roofline": None, "note": "sharded mode: see the default (replica) line for roofline and cpu_baseline"}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5", choices=["config1", "config2", "config3", "config5"])
    ap.add_argument("--fuse-pap", type=int, default=None, help="library options (include/nk.h); default: the library's")
    ap.add_argument("--pdl", type=int, default=None)
    ap.add_argument("--fuse-p", type=int, default=None)
    ap.add_argument("--fuse-gs", type=int, default=None)
    ap.add_argument("--graph", type=int, default=None)
    ap.add_argument("--coop", type=int, default=None)
    ap.add_argument("--defer-x", type=int, default=None)
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per ax_e launch from the committed ncu --set full capture (profiles/)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sharded", action="store_true",
                    help="partition ONE mesh over the ranks (distributed gs / CG) instead of N replicas")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return
    out = run_sharded(args) if args.sharded else run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
