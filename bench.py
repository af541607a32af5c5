#!/usr/bin/env python
"""bench.py -- headline benchmark of the vmg hot path (BASELINE.json metric: multigrid cell-updates/s and
solves/s at 4.19M cells fp64; % of B200 HBM BW).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 3|4|2|5]

A step = one pass of the whole hot path over one batch of synthetic input: vmg_set_coeffs (S0 coefficient
averaging + stencil build) + vmg_set_bc + vmg_solve from a zero guess to relative residual 1e-12 (S1 fold_bc,
S6 norms, ~10 V-cycles of S2-S5, S7 sequencing).  Workload at N = 1: BASELINE.json configs[2], the 256x128x128
(4 194 304-cell) electrostatic Poisson solve the metric is quoted on.  N > 1: independent replicas, one per
GPU, no collective on the data path (replicas only).

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
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

import numpy as np

# algorithmic bytes per cell: fp64, 6 input arrays + 1 output
B_SMOOTH_PASS = 56.0        # one blocked pass of nu sweeps: read phi,btilde,dinv,wx,wy,wz, write phi
B_RESID_RESTRICT = 49.0
B_PROLONG_CORRECT = 17.0
B_FOLD = 16.0
B_NORM = 8.0
B_SETCOEFFS = 24.0
# DRAM bytes that the dominant kernel class actually moved (roofline.traffic) come from an ncu capture, not from this
# run: profiles/traffic.json holds them per config together with the commit and a hash of the kernel sources they were
# captured at; when the sources have changed since, the entry is stale and the line carries null.
KERNEL_SOURCES = ("vmg_kernels.cuh", "vmg_sched.cuh", "vmg_api.cu", "vmg_internal.h")


def kernel_sources_sha():
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2507_08200_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def captured_traffic(config: int, opts):
    """(cold, warm, note) DRAM bytes per nu-sweep pass of the level-0 smoother from profiles/traffic.json, or Nones."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
        e = t[f"config{config}"]
        if opts or e["sources_sha16"] != kernel_sources_sha():
            return None, None, f"profiles/traffic.json entry is for sources {e['sources_sha16']} (commit {e['commit']}); the kernels changed since or options are set"
        return e["traffic_pass_cold"], e["traffic_pass_warm"], e["note"]
    except Exception as ex:   # no capture for this config
        return None, None, f"no ncu capture for this config in profiles/traffic.json ({type(ex).__name__})"


def level_cells(nx, ny, nz):
    """cells per level, finest first (R11: halve while all active dims are even and stay >= 2)."""
    three_d = nz > 1
    out = [nx * ny * nz]
    while nx % 2 == 0 and ny % 2 == 0 and nx // 2 >= 2 and ny // 2 >= 2 and (not three_d or (nz % 2 == 0 and nz // 2 >= 2)):
        nx, ny, nz = nx // 2, ny // 2, (nz // 2 if three_d else 1)
        out.append(nx * ny * nz)
    return out


def work_model(p, nu1=3, nu2=3, nbottom=32):
    cells = level_cells(p.nx, p.ny, p.nz)
    upper = sum(cells[:-1])
    return {
        "updates_per_cycle": (nu1 + nu2) * upper + nbottom * cells[-1],
        "bytes_per_cycle": (2 * B_SMOOTH_PASS + B_RESID_RESTRICT + B_PROLONG_CORRECT) * upper,
        "bytes_solve_fixed": (B_FOLD + B_NORM) * cells[0],
        "bytes_set_coeffs": B_SETCOEFFS * sum(cells),
        "cells": cells,
    }


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def max_over_ranks(seconds: float, dist, device=None) -> float:
    """Time of the slowest replica (the contract: barrier on both sides, MAX over ranks)."""
    if dist is None:
        return seconds
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_replicas(units_per_rank: float, seconds: float, world: int, dist, device=None) -> float:
    """Whole-job throughput of `world` independent replicas: every rank processes
    the same number of units, the job takes as long as its slowest rank; no collective touches the data path."""
    return world * units_per_rank / max_over_ranks(seconds, dist, device)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.01):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.max_mhz = index, period, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def finish(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2.0)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def make_problem(config: int):
    from paper_2507_08200_b200 import inputs
    return inputs.CONFIGS[config]()


# ----------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on the box's host cores
# ----------------------------------------------------------------------------------------------------
def oracle_sample(p, cycles_per_step: int):
    """A bounded sample of the workload: set_coeffs + set_bc + `cycles_per_step` V-cycles (rtol = 0) -- for config 3
    that is one whole step (the solve needs 10 cycles), ~25 core-seconds on the 16 host threads."""
    from oracle import Oracle
    t0 = time.perf_counter()
    o = Oracle.from_problem(p)
    o.solve(p.rhs, rtol=0.0, max_vcycles=cycles_per_step)
    dt = time.perf_counter() - t0
    o.close()
    return dt


def set_oracle_threads(n: int) -> bool:
    """OpenMP threads of the oracle library (it is the only OpenMP user in the process)."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_cycles(p):
    """V-cycles per oracle sample: a whole solve where that stays within seconds, 2 cycles at 512^3."""
    return 10 if p.ncells <= (1 << 23) else 2


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    p = make_problem(args.config)
    wm = work_model(p)
    cyc = oracle_cycles(p)
    for _ in range(args.warmup):
        oracle_sample(p, cyc)
    times = [oracle_sample(p, cyc) for _ in range(args.steps)]
    dt = float(np.mean(times))
    value = cyc * wm["updates_per_cycle"] / dt
    cores = os.cpu_count()
    sample = (f"set_coeffs + set_bc + {cyc} V(3,3)-cycles (rtol=0) of {p.name} per step, "
              f"OpenMP over all {cores} host threads, gcc -O2 -ffp-contract=off")
    line = {
        "impl": "reference", "metric": "multigrid_cell_updates_per_s", "value": value, "unit": "cell-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": p.name, "cells": p.ncells, "sample": sample},
        "vcycles_per_s": cyc / dt,
        "cpu_baseline": {"value": value, "unit": "cell-updates/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def timestep_leg(binding, torch, p, d, d_bc, dev, s, flush, nsteps: int = 3, rtol: float = 1e-10):
    """20 elliptic solves per (single-corrector) time step on the 256x128x128 grid, all through the public calls:
      Poisson        config 3 (a = 0, b = 1 passed as NULL, electrode Dirichlet values),
      15 species     alpha a phi - beta_k div(b grad phi) = f with config 4's a = n_e/dt, b = (5/3) D_e n_e and
                     beta_k = 15 diffusivity ratios over two decades (same arrays, different operator per species),
      energy         config 4 itself,
      3 x photoion.  a = 1 (array), alpha = (lambda_j p)^2 for three absorption lengths, b = 1 (NULL), random source.
    Right-hand sides grow by 1 % per step; every solve starts from its field of the previous step (PAPER.md:142-148:
    the correctors re-solve with slowly changing data).  Step 0 (cold start) is the warm-up."""
    from paper_2507_08200_b200 import inputs
    p4 = inputs.config4(p.ny)
    up = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(dev)
    d4 = {k: up(getattr(p4, k)) for k in ("a", "bx", "by", "bz", "rhs")}
    ones = torch.ones_like(d["rhs"])
    gen = torch.Generator(device=dev).manual_seed(1234)
    photo_rhs = torch.randn(d["rhs"].shape, generator=gen, device=dev, dtype=torch.float64)
    betas = np.logspace(-1.0, 1.0, 15)
    lambdas2 = [1.0e2, 1.0e3, 1.0e4]
    eqs = [("poisson", lambda: (s.set_coeffs(d["a"], None, None, None, p.alpha, p.beta), s.set_bc(p.bc_type, d_bc)), d["rhs"])]
    for b_k in betas:
        eqs.append(("species", lambda b_k=b_k: (s.set_coeffs(d4["a"], d4["bx"], d4["by"], d4["bz"], 1.0, float(b_k)), s.set_bc(p4.bc_type, None)), d4["rhs"]))
    eqs.append(("energy", lambda: (s.set_coeffs(d4["a"], d4["bx"], d4["by"], d4["bz"], 1.0, 1.0), s.set_bc(p4.bc_type, None)), d4["rhs"]))
    for l2 in lambdas2:
        eqs.append(("photo", lambda l2=l2: (s.set_coeffs(ones, None, None, None, l2, 1.0), s.set_bc(p4.bc_type, None)), photo_rhs))
    fields = [torch.zeros_like(d["rhs"]) for _ in eqs]
    times, cycles = [], []
    for step in range(nsteps + 1):
        scale = 1.0 + 0.01 * step
        flush.fill_(1.0)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ncyc = 0
        for (name, setup, rhs), phi in zip(eqs, fields):
            setup()
            st = s.solve(rhs * scale, phi, rtol=rtol, max_vcycles=50)
            assert st == 0, (name, st)
            ncyc += s.get_info()[0]
        e1.record()
        e1.synchronize()
        if step > 0:
            times.append(e0.elapsed_time(e1))
            cycles.append(ncyc)
    ms = float(np.mean(times))
    out = {"ms_per_time_step": ms, "time_steps_per_s": 1e3 / ms, "solves_per_time_step": len(eqs),
           "vcycles_per_time_step": float(np.mean(cycles)), "rtol": rtol,
           "sequence": "Poisson + 15 species + energy + 3 photoionisation; set_coeffs + set_bc + warm-started solve each; one handle"}

    # The same time step with the 16 transport solves (15 species + energy: independent of each other once the potential is
    # known) advanced together by vmg_solve_batch, one handle and one stream each (SURVEY.md 8(f) N1 inside N3: the
    # paper's "multi-component MG solves"); Poisson before them and the photoionisation solves after,
    # on the first handle as above.
    nb = 16
    streams = [torch.cuda.Stream() for _ in range(nb)]
    hs = [binding.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, stream=st) for st in streams]
    for hb in hs:
        hb.set_bc(p4.bc_type, None)
    tb = list(betas) + [1.0]
    bfields = [torch.zeros_like(d["rhs"]) for _ in range(nb)]
    for f in fields:
        f.zero_()
    times_b, cycles_b = [], []
    for step in range(nsteps + 1):
        scale = 1.0 + 0.01 * step
        flush.fill_(1.0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ncyc = 0
        name, setup, rhs = eqs[0]
        setup()
        assert s.solve(rhs * scale, fields[0], rtol=rtol, max_vcycles=50) == 0
        ncyc += s.get_info()[0]
        torch.cuda.synchronize()
        for hb, b_k in zip(hs, tb):
            hb.set_coeffs(d4["a"], d4["bx"], d4["by"], d4["bz"], 1.0, float(b_k))
        rb = d4["rhs"] * scale
        torch.cuda.synchronize()
        sts = binding.solve_batch(hs, [rb] * nb, bfields, rtol=rtol, max_vcycles=50)
        assert all(v == 0 for v in sts), sts
        ncyc += sum(hb.get_info()[0] for hb in hs)
        for (name, setup, rhs), phi in zip(eqs[17:], fields[17:]):
            setup()
            assert s.solve(rhs * scale, phi, rtol=rtol, max_vcycles=50) == 0
            ncyc += s.get_info()[0]
        torch.cuda.synchronize()
        if step > 0:
            times_b.append((time.perf_counter() - t0) * 1e3)
            cycles_b.append(ncyc)
    for hb in hs:
        hb.destroy()
    out["batched_transport"] = {"ms_per_time_step": float(np.mean(times_b)), "time_steps_per_s": 1e3 / float(np.mean(times_b)),
                                "vcycles_per_time_step": float(np.mean(cycles_b)), "handles": nb,
                                "timing": "host clock, device synchronised on both sides"}
    return out


# ----------------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------------
def amr_leg(binding, torch, dev, flush, ny: int, steps: int = 5, with_oracle: bool = True, patches: int = 1, opts=()):
    """Two-level composite solve (second half): config 3 with the streamer head
    refined -- the 2 ny x ny x ny box plus a patch of ny x ny/2 x ny/2 fine cells -- through vmg_amr_*; explicit arrays of
    ones on both levels as in the headline run.  patches = 3: three heads side by side, a patch around each.  Device-resident
    inputs, CUDA events on the solver's stream, L2 flushed between solves.  The oracle (oracle/amr_oracle.c) is timed beside
    it on ONE solve."""
    from paper_2507_08200_b200 import inputs
    p = inputs.amr_streamer(ny) if patches == 1 else inputs.amr_streamers(ny)
    c = p.coarse
    up = lambda x: None if x is None else torch.from_numpy(np.ascontiguousarray(x)).to(dev)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        s = binding.VmgAmr(c.nx, c.ny, c.nz, c.dx, c.dy, c.dz, p.lo, p.hi, stream=stream)
        for kv in opts:
            key, val = kv.split("=")
            s.set_option(key, float(val))
        coarse = [up(x) for x in p.coarse_coeffs()]
        fine = [[up(x) for x in f] for f in p.fine_coeffs()] if p.multi else [up(x) for x in p.fine_coeffs()]
        bc = [up(v) for v in c.bc_value]
        rhs_c = up(c.rhs)
        rhs_f = [up(r) for r in p.rhs_f] if p.multi else up(p.rhs_f)
        phi_c = torch.zeros_like(rhs_c)
        phi_f = [torch.zeros_like(r) for r in rhs_f] if p.multi else torch.zeros_like(rhs_f)
        s.set_coeffs(coarse, fine, c.alpha, c.beta)
        s.set_bc(c.bc_type, bc)
        times, cyc, st, rr = [], 0, 0, 0.0
        for it in range(steps + 2):
            phi_c.zero_()
            for t in (phi_f if p.multi else [phi_f]):
                t.zero_()
            flush.fill_(1.0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            _, _, st, cyc, rr, hist = s.solve(rhs_c, rhs_f, phi_c, phi_f, rtol=p.rtol, max_cycles=p.max_cycles)
            e1.record(stream)
            e1.synchronize()
            assert st == 0, f"composite solve status {st}"
            if it >= 2:
                times.append(e0.elapsed_time(e1) * 1e-3)
        launches = s.last_launch_count()
    stream.synchronize()
    dims = p.fine_dims if p.multi else [p.fine_dims]
    nf = int(sum(np.prod(d) for d in dims))
    out = {"workload": p.name, "coarse_cells": c.ncells, "fine_cells": nf, "patches": len(dims),
           "solve_ms": float(np.mean(times)) * 1e3,
           "solves_per_s": 1.0 / float(np.mean(times)), "cycles": cyc, "ms_per_cycle": float(np.mean(times)) * 1e3 / max(cyc, 1),
           "relres": rr, "launches_per_solve": int(launches), "nu_f": 6,
           "cycle": "composite residual -> one V(3,3) cycle of the box -> correction -> 6 red-black sweeps on every patch"}
    if with_oracle:
        from oracle import AmrOracle
        o = AmrOracle(c.nx, c.ny, c.nz, c.dx, c.dy, c.dz, p.lo, p.hi)
        o.set_coeffs(p.coarse_coeffs(), p.fine_coeffs(), c.alpha, c.beta)
        o.set_bc(c.bc_type, c.bc_value)
        t0 = time.perf_counter()
        r = o.solve(c.rhs, p.rhs_f, rtol=p.rtol, max_cycles=p.max_cycles)
        dt = time.perf_counter() - t0
        gf, of = (phi_f if p.multi else [phi_f]), (r[1] if p.multi else [r[1]])
        err = max([float(np.abs(phi_c.cpu().numpy() - r[0]).max())] + [float(np.abs(g.cpu().numpy() - w).max()) for g, w in zip(gf, of)])
        out["oracle"] = {"solve_s": dt, "cycles": r[3], "cores": os.cpu_count(), "rel_linf_gpu_vs_oracle": err / float(np.abs(r[0]).max())}
    s.destroy()
    return out


def run_vmg(args):
    import torch
    from paper_2507_08200_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; --impl reference times the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    p = make_problem(args.config)
    wm = work_model(p)
    peak, peak_src = measured_peak_gbs()
    stream = torch.cuda.Stream()
    dev = torch.device("cuda", local)

    # host copies in pinned memory (for the e2e leg), device-resident copies (for the headline leg)
    host = {k: (None if v is None else torch.from_numpy(np.ascontiguousarray(v)).pin_memory())
            for k, v in dict(a=p.a, bx=p.bx, by=p.by, bz=p.bz, rhs=p.rhs).items()}
    host_bc = [None if v is None else torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for v in p.bc_value]
    host_phi = torch.zeros(p.rhs.shape, dtype=torch.float64).pin_memory()
    with torch.cuda.stream(stream):
        d = {k: (None if v is None else v.to(dev, non_blocking=True)) for k, v in host.items()}
        d_bc = [None if v is None else v.to(dev, non_blocking=True) for v in host_bc]
        phi = torch.zeros(p.rhs.shape, dtype=torch.float64, device=dev)
        flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)   # 256 MiB > 126 MB L2
        s = binding.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, stream=stream)
        for kv in args.opt:
            key, val = kv.split("=")
            s.set_option(key, float(val))
    stream.synchronize()

    def step_resident():
        """inputs already resident in HBM"""
        phi.zero_()
        s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
        s.set_bc(p.bc_type, d_bc)
        return s.solve(d["rhs"], phi, rtol=p.rtol, max_vcycles=p.max_vcycles)

    side = torch.cuda.Stream()

    def step_e2e():
        """host buffers in, host buffer out: H2D of every input and D2H of phi inside the timed region.  The coefficient
        arrays go first on the solver's stream, rhs and the initial guess on a second stream, so that vmg_set_coeffs /
        vmg_set_bc (enqueue-only on a caller's stream) run while the last 67 MB are still crossing PCIe; the 236 MB at the
        link's ~55 GB/s remain the floor of this leg."""
        dd = {k: (None if v is None else v.to(dev, non_blocking=True)) for k, v in host.items() if k != "rhs"}
        dbc = [None if v is None else v.to(dev, non_blocking=True) for v in host_bc]
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            rhs_d = host["rhs"].to(dev, non_blocking=True)
            ph = host_phi.to(dev, non_blocking=True)                   # zero initial guess from the host
            rhs_d.record_stream(stream); ph.record_stream(stream)
        s.set_coeffs(dd["a"], dd["bx"], dd["by"], dd["bz"], p.alpha, p.beta)
        s.set_bc(p.bc_type, dbc)
        stream.wait_stream(side)
        st = s.solve(rhs_d, ph, rtol=p.rtol, max_vcycles=p.max_vcycles)
        out_host.copy_(ph, non_blocking=True)
        return st

    out_host = torch.empty(p.rhs.shape, dtype=torch.float64).pin_memory()
    h2d = sum(v.numel() * 8 for v in host.values() if v is not None) + sum(v.numel() * 8 for v in host_bc if v is not None) \
        + host_phi.numel() * 8
    d2h = out_host.numel() * 8

    def timed(fn, steps, warmup, sampler=None, after_warmup=None):
        times, cycles, launches = [], [], 0
        with torch.cuda.stream(stream):
            for _ in range(warmup):
                fn()
            stream.synchronize()
            if after_warmup is not None:
                after_warmup()
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()
            if sampler is not None:
                sampler.start()
            for _ in range(steps):
                flush.fill_(1.0)                                   # evict L2 between timed iterations
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                l0 = s.total_launch_count()
                e0.record(stream)
                st = fn()
                e1.record(stream)
                e1.synchronize()
                assert st in (0, 1), f"solve status {st}"
                times.append(e0.elapsed_time(e1) * 1e-3)
                cycles.append(s.get_info()[0])
                launches += s.total_launch_count() - l0
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
        return np.array(times), np.array(cycles), launches

    sampler = ClockSampler(local)
    times, cycles, launches = timed(step_resident, args.steps, args.warmup, sampler)
    total = max_over_ranks(float(times.sum()), dist, dev)
    updates_per_step = float(np.mean(cycles)) * wm["updates_per_cycle"]
    value = aggregate_replicas(args.steps * updates_per_step, float(times.sum()), world, dist, dev)

    # solve-only and per-kernel-class numbers (plain launches with event pairs; same workload)
    s.set_option("profile", 1)
    ptimes, pcycles, _ = timed(step_resident, max(2, min(args.steps, 5)), 1, after_warmup=lambda: s.set_option("profile", 1))
    prof = s.get_profile()
    s.set_option("profile", 0)
    n_prof_cycles = float(pcycles.sum())
    sm_ms, sm_launches = prof["smooth_l0"]
    n0 = wm["cells"][0]
    achieved = (2 * B_SMOOTH_PASS * n0 * n_prof_cycles) / (sm_ms * 1e-3) / 1e9 if sm_ms > 0 else 0.0
    klass = {k: {"ms_per_cycle": v[0] / max(n_prof_cycles, 1), "launches_per_cycle": v[1] / max(n_prof_cycles, 1)}
             for k, v in prof.items()}

    # solve only (coefficients already set): the SURVEY's solves/s definition
    def solve_only():
        phi.zero_()
        return s.solve(d["rhs"], phi, rtol=p.rtol, max_vcycles=p.max_vcycles)
    stimes, scycles, _ = timed(solve_only, args.steps, 1)
    solve_s = float(np.mean(stimes))
    ncyc = float(np.mean(scycles))
    bytes_solve = ncyc * wm["bytes_per_cycle"] + wm["bytes_solve_fixed"]
    traffic_cold, traffic_warm, traffic_note = captured_traffic(args.config, args.opt)

    # MG-preconditioned conjugate gradients: the same solve through vmg_solve_pcg
    def solve_pcg_only():
        phi.zero_()
        return s.solve_pcg(d["rhs"], phi, rtol=p.rtol if p.rtol > 0 else 1e-12, max_iter=max(p.max_vcycles, 60))
    ptimes_, piters, _ = timed(solve_pcg_only, max(2, min(args.steps, 5)), 1)
    pcg = {"solve_ms": float(np.mean(ptimes_)) * 1e3, "solves_per_s": world / float(np.mean(ptimes_)), "iterations": float(np.mean(piters)),
           "relres": s.get_info()[1], "note": "one symmetric V-cycle, one operator application and two dot products per iteration"}

    # constant face weights: the same solve with b == NULL (b = 1: the Poisson equation itself, Eq. 3), which
    # selects the kernels that do not load the weight arrays; bitwise the same phi (tests).  Only where b is all ones.
    const_w = None
    if all(float(d[k].min()) == 1.0 and float(d[k].max()) == 1.0 for k in ("bx", "by", "bz") if d[k] is not None):
        s.set_coeffs(d["a"], None, None, None, p.alpha, p.beta)
        ctimes, ccycles, _ = timed(solve_only, max(2, min(args.steps, 5)), 1)
        const_w = {"solve_ms": float(np.mean(ctimes)) * 1e3, "solves_per_s": world / float(np.mean(ctimes)),
                   "cycles": float(np.mean(ccycles)), "us_per_vcycle": float(np.mean(ctimes)) / float(np.mean(ccycles)) * 1e6,
                   "note": "vmg_set_coeffs with b == NULL; not the headline (the roofline run reads explicit arrays of ones)"}
        s.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)

    # batched multi-component solves (the paper's own optimisation): K independent
    # solves of the same workload, one handle and one stream each, advanced in lock-step by vmg_solve_batch
    batched = None
    if args.batch > 1:
        K = args.batch
        bstreams = [torch.cuda.Stream() for _ in range(K)]
        bsolvers, bphis = [], []
        for st_ in bstreams:
            with torch.cuda.stream(st_):
                sv = binding.Vmg(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, stream=st_)
                for kv in args.opt:
                    key, val = kv.split("=")
                    sv.set_option(key, float(val))
                sv.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
                sv.set_bc(p.bc_type, d_bc)
                bphis.append(torch.zeros(p.rhs.shape, dtype=torch.float64, device=dev))
            bsolvers.append(sv)
        torch.cuda.synchronize()
        btimes = []
        for it in range(1 + max(2, min(args.steps, 5))):
            for ph in bphis:
                ph.zero_()
            flush.fill_(1.0)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sts = binding.solve_batch(bsolvers, [d["rhs"]] * K, bphis, rtol=p.rtol, max_vcycles=p.max_vcycles)
            torch.cuda.synchronize()
            if it > 0:
                btimes.append(time.perf_counter() - t0)
        bcyc = float(np.mean([sv.get_info()[0] for sv in bsolvers]))
        bt = float(np.mean(btimes))
        batched = {"k": K, "solves_per_s": world * K / bt, "vcycles_per_s": world * K * bcyc / bt, "ms_per_batch": bt * 1e3,
                   "hbm_frac": K * (bcyc * wm["bytes_per_cycle"] + wm["bytes_solve_fixed"]) / bt / 1e9 / peak,
                   "timing": "host clock around vmg_solve_batch, device synchronised on both sides", "statuses": sorted(set(sts))}
        for sv in bsolvers:
            sv.destroy()
        # the same K solves with KERNEL-LEVEL batching (vmg_create_batch: one allocation, one stream; the coarser levels of all
        # K problems as single launches over planes x problems, K CTAs in the tail; level 0 one problem at a time at this size)
        with torch.cuda.stream(stream):
            gs = binding.create_batch(K, p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, stream=stream)
            for sv in gs:
                for kv in args.opt:
                    key, val = kv.split("=")
                    sv.set_option(key, float(val))
                sv.set_coeffs(d["a"], d["bx"], d["by"], d["bz"], p.alpha, p.beta)
                sv.set_bc(p.bc_type, d_bc)
            gtimes = []
            for it in range(1 + max(2, min(args.steps, 5))):
                for ph in bphis:
                    ph.zero_()
                flush.fill_(1.0)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                gsts = binding.solve_batch(gs, [d["rhs"]] * K, bphis, rtol=p.rtol, max_vcycles=p.max_vcycles)
                torch.cuda.synchronize()
                if it > 0:
                    gtimes.append(time.perf_counter() - t0)
            gt = float(np.mean(gtimes))
            batched["kernel_level"] = {"solves_per_s": world * K / gt, "ms_per_batch": gt * 1e3, "statuses": sorted(set(gsts)),
                                       "hbm_frac": K * (bcyc * wm["bytes_per_cycle"] + wm["bytes_solve_fixed"]) / gt / 1e9 / peak,
                                       "note": "vmg_create_batch group; at this size level 0 runs one problem at a time (L2 reuse), levels 1.. problem-major"}
            for sv in gs:
                sv.destroy()

    # one time step of the paper's scheme (Eq. 9-10): Poisson, 15
    # species, electron energy and three photoionisation Helmholtz solves, each vmg_set_coeffs + vmg_set_bc +
    # vmg_solve on ONE handle, warm-started from the previous step's field while the data drift by 1 % per step
    timestep = None
    if args.config == 3 and not args.no_timestep:
        timestep = timestep_leg(binding, torch, p, d, d_bc, dev, s, flush)
    amr = None
    if args.config == 3 and not args.no_amr and world == 1:
        amr = amr_leg(binding, torch, dev, flush, p.ny, with_oracle=not args.no_cpu_baseline)
        amr["three_patches"] = amr_leg(binding, torch, dev, flush, p.ny, steps=3, with_oracle=not args.no_cpu_baseline, patches=3)

    # end to end through the C-ABI with host buffers
    etimes, ecycles, _ = timed(step_e2e, args.steps, max(1, min(args.warmup, 2)))
    etotal = max_over_ranks(float(etimes.sum()), dist, dev)
    e2e_value = world * args.steps * float(np.mean(ecycles)) * wm["updates_per_cycle"] / etotal
    clocks = sampler.finish()   # sampled over all timed regions of this run (headline, per-kernel, solve-only, end-to-end)

    line = {
        "metric": "multigrid_cell_updates_per_s", "value": value, "unit": "cell-updates/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": p.name, "cells": p.ncells, "levels": len(wm["cells"]), "smoother": "V(3,3) red-black GS",
                   "rtol": p.rtol, "cycles_per_solve": ncyc, "step": "vmg_set_coeffs + vmg_set_bc + vmg_solve",
                   "l2": "256 MiB flush write between timed steps; level-0 working set 201 MB > 126 MB L2",
                   "multi_gpu": "replicas only", "options": args.opt},
        "solves_per_s": world / solve_s, "vcycles_per_s": world * ncyc / solve_s,
        "solve_ms": solve_s * 1e3,
        "hbm_frac_solve": bytes_solve / solve_s / 1e9 / peak,
        "hbm_frac_note": f"algorithmic bytes (203.4 B/cell/V-cycle model) / solve time / {peak} GB/s {peak_src}",
        "roofline": {"bound": "hbm", "kernel": "level-0 red-black smoother (all launches of a nu-sweep pass)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "achieved_mode": "event pairs around the plain launches of the class (option profile=1: host-driven loop, no graph), "
                                      "in a second region right after the timed one; inside the graph the same launches are ~8 % faster",
                     "traffic": traffic_cold, "traffic_warm": traffic_warm, "traffic_note": traffic_note,
                     "achieved_bytes_per_pass": B_SMOOTH_PASS * n0, "peak_source": peak_src,
                     "launches_per_pass": sm_launches / max(2 * n_prof_cycles, 1),
                     # the number the target is stated on (north_star: ">= 60 % ... across the V-cycle"): whole solve, graph mode
                     "cycle_frac": bytes_solve / solve_s / 1e9 / peak, "cycle_us": solve_s / ncyc * 1e6,
                     "cycle_bytes": wm["bytes_per_cycle"],
                     "cycle_note": "algorithmic bytes of the whole solve (203.4 B/cell/V-cycle, SURVEY 8(d)) / event-timed vmg_solve in its default mode"},
        "kernel_classes": klass,
        "pcg": pcg,
        "const_weights": const_w,
        "batched": batched,
        "timestep": timestep,
        "amr": amr,
        "e2e": {"value": e2e_value, "unit": "cell-updates/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": etotal / args.steps * 1e3},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cyc = oracle_cycles(p)
        oracle_sample(p, 1)
        t_or = [oracle_sample(p, cyc) for _ in range(2)]
        dt = float(np.mean(t_or))
        line["cpu_baseline"] = {"value": cyc * wm["updates_per_cycle"] / dt, "unit": "cell-updates/s",
                                "cores": os.cpu_count(), "kind": "oracle", "cpu": cpu_model(),
                                "sample": f"set_coeffs + set_bc + {cyc} V(3,3)-cycles of {p.name}, mean of 2 runs"}
        # the same oracle on ONE thread (SURVEY 8(d) "(a) single thread"): the figure comparable with the paper's
        # "1 GPU vs 1 CPU core" ratio; bounded to 2 cycles
        if set_oracle_threads(1):
            c1 = 2 if p.ncells <= (1 << 23) else 1
            dt1 = oracle_sample(p, c1)
            set_oracle_threads(os.cpu_count())
            v1 = c1 * wm["updates_per_cycle"] / dt1
            line["cpu_baseline"]["single_thread"] = {
                "value": v1, "unit": "cell-updates/s", "cores": 1,
                "sample": f"set_coeffs + set_bc + {c1} V(3,3)-cycles of {p.name}, one run",
                "gpu_over_one_core": value / v1,
                "paper_context": "the paper reports ~150-400x per TIME STEP for 1 GPU (H100/A100/MI250X) vs 1 CPU core at 4 M cells, 15 species (PAPER.md:16, 305-307): context, not the target"}
    s.destroy()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def write_traffic_json(args):
    """profiles/traffic.json from two ncu launch lists of the default path (`--metrics dram__bytes_read.sum,
    dram__bytes_write.sum,gpu__time_duration.sum`; cold = ncu's default cache control, warm = --cache-control none):
    DRAM bytes of the level-0 half-sweep launches, per nu-sweep pass of 6 launches, stamped with the commit and the hash of
    the kernel sources so that a later bench run can tell whether the entry still describes the code it times."""
    import csv
    import subprocess
    p = make_problem(args.config)

    def per_launch(path):
        per = {}
        with open(path) as f:
            rows = [r for r in csv.reader(f) if len(r) > 10]
        hdr = rows[0]
        ik, im, iv, ig, iid = (hdr.index(k) for k in ("Kernel Name", "Metric Name", "Metric Value", "Grid Size", "ID"))
        for r in rows[1:]:
            if "smooth_colour_kernel" in r[ik] and r[ig].replace(" ", "") == f"(1,{p.ny // 2},{p.nz})":
                per.setdefault(r[iid], {})[r[im]] = float(r[iv].replace(",", ""))
        vals = [v["dram__bytes_read.sum"] + v["dram__bytes_write.sum"] for v in per.values()]
        us = [v["gpu__time_duration.sum"] / 1e3 for v in per.values()]
        return float(np.mean(vals)), float(np.mean(us)), len(vals)

    cold, cold_us, n_c = per_launch(args.traffic_from[0])
    warm, warm_us, n_w = per_launch(args.traffic_from[1])
    head = subprocess.run(["git", "rev-parse", "--short=12", "HEAD"], cwd=ROOT, capture_output=True, text=True).stdout.strip()
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as f:
            t = json.load(f)
    except Exception:
        t = {}
    t[f"config{args.config}"] = {
        "workload": p.name, "commit": head, "sources_sha16": kernel_sources_sha(), "sources": list(KERNEL_SOURCES),
        "traffic_pass_cold": 6 * cold, "traffic_pass_warm": 6 * warm,
        "per_launch": {"cold_bytes": cold, "cold_us": cold_us, "cold_launches": n_c, "warm_bytes": warm, "warm_us": warm_us, "warm_launches": n_w},
        "note": "DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum, ncu) of the six level-0 half-sweep launches of one nu = 3 pass; "
                "cold = every launch alone with flushed caches, warm = the L2 as the previous launch left it (--cache-control none); "
                "algorithmic 234.9 MB per pass; commands in profiles/r2_dram.md"}
    with open(path, "w") as f:
        json.dump(t, f, indent=1)
        f.write("\n")
    print(json.dumps(t[f"config{args.config}"]))


def run_blocked_probe(args):
    """Profiling aid (not a bench line): the level-0 strokes of the configured workload through the temporally blocked
    smoother passes (vmg_set_option blocked = 1 | 2 | 3) as separate calls, so that `ncu -k regex:smooth_block` sees the
    pass kernels alone.  Prints what it ran; times come from ncu (profiles/)."""
    import torch
    from paper_2507_08200_b200 import binding
    p = make_problem(args.config)
    s, d = binding.from_problem(p)
    s.set_option("blocked", args.blocked_probe)
    gen = torch.Generator(device="cuda").manual_seed(7)
    phi = torch.randn(p.rhs.shape, generator=gen, device="cuda", dtype=torch.float64)
    e = torch.randn(tuple(n // 2 for n in p.rhs.shape), generator=gen, device="cuda", dtype=torch.float64)
    for _ in range(max(1, args.steps)):
        s.step_smooth(0, phi, d["rhs"], 3)          # two passes of S = 3
        s.step_down(0, phi, d["rhs"])               # S = 3, then S = 3 + residual and restriction
        s.step_up(0, phi, d["rhs"], e)              # prolongation + S = 3, then S = 3
    torch.cuda.synchronize()
    print(json.dumps({"probe": "blocked_passes", "blocked": args.blocked_probe, "workload": p.name, "repeats": max(1, args.steps),
                      "calls": ["step_smooth(level 0, 3 sweeps)", "step_down(level 0)", "step_up(level 0)"]}), flush=True)
    s.destroy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="vmg", choices=["vmg", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[2, 3, 4, 5])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-timestep", action="store_true", help="skip the per-time-step sequence leg")
    ap.add_argument("--no-amr", action="store_true", help="skip the two-level composite (AMR) leg")
    ap.add_argument("--amr-only", action="store_true",
                    help="profiling aid: run only the composite (AMR) leg (--steps solves after 2 untimed ones), print its JSON and exit")
    ap.add_argument("--batch", type=int, default=8, help="K for the batched multi-component leg (0/1: skip)")
    ap.add_argument("--opt", action="append", default=[], help="vmg_set_option key=value (experiments)")
    ap.add_argument("--traffic-from", nargs=2, metavar=("COLD_CSV", "WARM_CSV"),
                    help="write profiles/traffic.json from two ncu launch lists (no GPU needed) and exit")
    ap.add_argument("--blocked-probe", type=int, default=0, choices=[0, 1, 2, 3],
                    help="profiling aid: run the level-0 strokes through the blocked passes of this kind and exit")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "vmg" else args.warmup
    if args.traffic_from:
        write_traffic_json(args)
    elif args.blocked_probe:
        run_blocked_probe(args)
    elif args.amr_only:
        import torch
        from paper_2507_08200_b200 import binding
        torch.cuda.set_device(0)
        dev = torch.device("cuda", 0)
        flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)
        out = amr_leg(binding, torch, dev, flush, 128, steps=args.steps, with_oracle=False, opts=args.opt)
        out["three_patches"] = amr_leg(binding, torch, dev, flush, 128, steps=args.steps, with_oracle=False, patches=3, opts=args.opt)
        print(json.dumps({"amr": out}))
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_vmg(args)


if __name__ == "__main__":
    main()
