#!/usr/bin/env python
"""bench.py -- throughput of the bound-motor microscale hot path (libmm, sm_100a) on BASELINE.json's configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cuda|reference] [--config i] [--fuse-t T]

One "step" = one macro step of the whole hot path on one workload of
BASELINE.json `configs`: mm_set_filament_velocity, then n_sub explicit substeps with the moment reduction at
the config's cadence (configs[3-4]: 50 substeps, moments every 10).  The density stays resident on the GPU
between steps, as the paper prescribes; step k+1 continues from step k's state.

Prints ONE JSON line (rank 0).  `value` = motor-cell updates/s (G/s), whole job, inputs resident in HBM;
`e2e` = same metric through the same C-ABI calls with pinned HOST buffers for (U,V,Omega) and the moments,
i.e. the host<->device copies of every macro step inside the timed region.  `roofline` is for the dominant
kernel (the fused advect+react(+moments) substep kernel), timed live with CUDA events on the library's stream: it is
bound by FMA issue ("alu"; peak = mm_measure_fma_peak in the same run); `roofline_hbm` is its HBM side (real DRAM rate of
the fused pass, the algorithmic rate, the unfused T = 1 point, each also against the nominal 8 TB/s).  `per_config`
holds short runs of the other single-GPU workloads of BASELINE.json (default run only).
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import mm_inputs as mi

METRIC = "motor_cell_updates_per_s"
UNIT = "G cell-updates/s"
ES = {"f64": 8, "f32": 4}


# --------------------------------------------------------------------------------------------- helpers
def measured_peaks():
    """HBM peak (GB/s) from the driver-written MEASURED_PEAKS.json, else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML; nvidia-smi as a fallback)."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80, "sync_boost": 0x10, "app_clocks": 0x2, "idle": 0x1}

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _once(self):
        if self._nv is not None:
            nv = self._nv
            self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
            try:
                bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
            except Exception:
                bits = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
            for name, bit in {**self.BAD, **self.NOTE}.items():
                if bits & bit and name != "idle":
                    self.reasons.add(name)
        else:
            import subprocess
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", "--query-gpu=clocks.sm,clocks.max.sm,"
                                  "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                                  "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap",
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True).stdout.strip()
            f = [x.strip() for x in out.split(",")]
            if len(f) >= 6:
                self.samples.append(float(f[0]))
                self.max_mhz = float(f[1])
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                    if v == "Active":
                        self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            self._stop.wait(0.05 if self._nv is not None else 0.2)

    def start(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def pick_workload(idx, free_bytes=None):
    """BASELINE.json north_star quotes the target 'at the largest config, on one GPU': configs[4] when its two
    density buffers fit, else the largest that does."""
    if idx is not None:
        return idx
    order = [4, 3, 1, 0]
    for i in order:
        w = mi.CONFIGS[i]
        need = 2 * w.grid.cells * ES[w.dtype] + (2 << 30)
        if free_bytes is None or need <= free_bytes:
            return i
    return 0


def rank_workload(w: mi.Workload, rank: int):
    """Weak scaling: configurations never interact, so rank r runs its own copy of the workload
    grid -- the r-th x-slab of a world-times-larger periodic domain -- drawn from seed + r.  No data-path collective."""
    from paper_1908_04279_b200 import shard
    return mi.Workload(w.name, w.grid, w.dtype, w.n_sub, w.moments_every, w.omega_max, shard.rank_seed(w.seed, rank),
                       w.params)


def with_scheme(w: mi.Workload, scheme: str):
    """--scheme rk2: the same workload advanced by the paper's RK2 + Superbee-in-s scheme (SURVEY.md 8(f) NEXT-1,
    MM_FLAG_RK2_SUPERBEE) instead of forward Euler + first-order upwind."""
    if scheme != "rk2":
        return w
    import dataclasses
    params = dataclasses.replace(w.params, flags=w.params.flags | mi.FLAG_RK2_SUPERBEE)
    return mi.Workload(w.name + "+rk2_superbee", w.grid, w.dtype, w.n_sub, w.moments_every, w.omega_max, w.seed, params)


def upload_inputs(mm, w, chunk_configs=2048, log=None):
    """S11 inputs for the whole workload, generated on the host in chunks of configurations and uploaded."""
    npdt = np.float64 if w.dtype == "f64" else np.float32
    g = w.grid
    st = mi.Stream(g, w.params.R, w.seed, w.omega_max)
    U, V, Om = st.velocities(npdt)
    buf = np.empty((min(chunk_configs, g.nc), g.ns, g.nxi, g.neta), npdt)
    t0 = time.time()
    for c0 in range(0, g.nc, chunk_configs):
        n = min(chunk_configs, g.nc - c0)
        st.density(n, npdt, out=buf[:n])
        mm.set_density_range(c0, n, buf[:n])
    st.close()
    if log:
        log(f"inputs: {g.cells/1e9:.2f} G cells generated+uploaded in {time.time()-t0:.1f} s")


# --------------------------------------------------------------------------------------------- CUDA arm
FMA_PER_CELL_UPDATE = 6     # S7 in coefficient form: self + s-upwind + four offset neighbours
NOMINAL_HBM_GBS = 8000.0    # north_star's "~8 TB/s"


def kernel_evidence(idx, kname):
    """DRAM bytes per launch and executed instructions per cell-update of this kernel family on this workload, from the
    committed `ncu --set full` captures (profiles/traffic.json); None where no capture of THIS kernel exists."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tr = json.load(f).get(f"configs[{idx}]", {}).get(kname.split("<")[0])
    except Exception:
        tr = None
    return tr or {}


def measure(mm, w, idx, args, steps, warmup, dev, stream, world, log, full_protocol):
    """Time `steps` macro steps of workload w on the context mm (density already uploaded).  Returns the pieces of the
    JSON line: value, e2e, rooflines, launches, clocks."""
    import torch
    from paper_1908_04279_b200 import binding as b, shard

    g, es = w.grid, ES[w.dtype]
    Uh, Vh, Oh = mi.Stream(g, w.params.R, w.seed, w.omega_max).velocities(np.float64 if w.dtype == "f64" else np.float32)
    n_mom = w.n_sub // w.moments_every
    Ud, Vd, Od = (torch.from_numpy(x).to(dev) for x in (Uh, Vh, Oh))          # device-resident inputs for `value`
    Fd = torch.empty((n_mom, g.nc, 2), dtype=torch.float64, device=dev)
    Td = torch.empty((n_mom, g.nc), dtype=torch.float64, device=dev)
    Up, Vp, Op = (torch.from_numpy(x).pin_memory() for x in (Uh, Vh, Oh))      # pinned host buffers for `e2e`
    Fp = torch.empty((n_mom, g.nc, 2), dtype=torch.float64).pin_memory()
    Tp = torch.empty((n_mom, g.nc), dtype=torch.float64).pin_memory()
    sub_events = []   # (start, stop, n_sub) around every mm_substep call of the timed region

    if args.full and full_protocol:   # the whole microscale step of Alg. 2 on this path: NEXT-2 + A0-A4 + NEXT-4
        psi_full = torch.rand(g.nc, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(7))
        mm.set_psi(psi_full)
        F2_full = torch.empty((g.nx, g.ny, 2), dtype=torch.float64, device=dev)
    full = args.full and full_protocol
    local_dt = args.local_dt and full_protocol

    def step(U, V, Om, F, T, record=False):
        mm.set_filament_velocity(U, V, Om)                                  # A0
        for k in range(n_mom):
            if full:
                mm.update_free_motors(None, None)                           # NEXT-2: M_b,coarse, cap, M_f
            if record:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                lc0 = mm.launch_count
            if local_dt:   # NEXT-3: same macro interval, every configuration with its own local steps
                mm.advance_local(w.moments_every * w.dt, args.cfl)
            else:
                mm.substep(w.moments_every, w.dt)                           # A1-A3 (+A4 fused into the last pass)
            if record:
                e1.record(stream)
                sub_events.append((e0, e1, w.moments_every, mm.launch_count - lc0))
            mm.moments(F[k], T[k])                                          # A4
            if full:
                mm.spread_force(F2_full)                                    # NEXT-4: Eq. 10

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps, U, V, Om, F, T, record=False):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = mm.launch_count
        e0.record(stream)
        for _ in range(nsteps):
            step(U, V, Om, F, T, record)
        e1.record(stream)
        barrier()
        return shard.max_over_ranks(e0.elapsed_time(e1), dev), mm.launch_count - l0

    # ---- warm-up, then the timed region (inputs resident in HBM)
    for _ in range(max(warmup, 0)):
        step(Ud, Vd, Od, Fd, Td)
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ else dev.index)
    sampler.start()
    ms, launches = timed(steps, Ud, Vd, Od, Fd, Td, record=True)
    clocks = sampler.stop()
    kname = mm.kernel_name
    units_rank_step = g.cells * w.n_sub          # cell-updates one rank performs per step
    local_info = None
    if local_dt:
        n_c = torch.empty(g.nc, dtype=torch.int32, device=dev)
        mm.local_steps(n_c, None)
        n_sum, n_max = int(n_c.sum().item()), int(n_c.max().item())
        units_rank_step = g.inner * n_sum * n_mom
        local_info = {"macro_dt": w.moments_every * w.dt, "cfl": args.cfl, "n_c_mean": round(n_sum / g.nc, 3),
                      "n_c_max": n_max, "n_c_min": int(n_c.min().item()),
                      "global_step_equivalent": round(g.cells * w.n_sub * world * steps / (ms * 1e-3) / 1e9, 2),
                      "note": "value counts the cell-updates actually performed (sum of n_c); global_step_equivalent "
                              "= rate at which the same physical time would need the global-dt substeps"}
    updates_per_step = units_rank_step * world
    value = shard.whole_job_rate(units_rank_step, steps, world, ms) / 1e9

    # ---- dominant kernel: average launch duration over the timed region (CUDA events on the library's stream)
    sub_ms = sum(a.elapsed_time(c) for a, c, _, _ in sub_events)
    sub_n = sum(n for _, _, n, _ in sub_events)
    fuse_opt = mm.get_option(b.MM_OPT_FUSE_T)
    m = __import__("re").search(r"T(?:<=|=)(\d+)", kname)
    fuse_t = 1 if args.scheme == "rk2" else (int(m.group(1)) if m else fuse_opt)   # depth of the launches actually made
    # launches of the pass kernel: counted by the library (local-step mode adds one rate + list kernel per pass: the
    # full-density passes are ceil(n_c_max / depth) per call)
    n_launch = sum(l for _, _, _, l in sub_events)
    if local_dt:
        n_launch = -(-local_info["n_c_max"] // max(fuse_t, 1)) * len(sub_events)
    cell_updates = float(g.cells) * sub_n if not local_dt else float(units_rank_step) / n_mom * len(sub_events)
    sub_s = sub_ms * 1e-3
    ev = kernel_evidence(idx, kname)
    # (1) the roof the fused kernel sits under: FMA issue (no tensor cores: 7-point stencil + reduction)
    fma_peak = b.measure_fma_peak(w.dtype, stream.cuda_stream)             # TFLOP/s, register-only probe, this run
    fma_fresh3 = b.measure_fma_rate(w.dtype, 3, stream.cuda_stream)        # ... with three fresh register operands per FMA
    nominal_fma = 148 * (64 if w.dtype == "f64" else 128) * 2 * 1.965e9 / 1e12
    alu_tflops = 2.0 * FMA_PER_CELL_UPDATE * cell_updates / sub_s / 1e12
    roofline = {"bound": "alu", "kernel": kname, "achieved": round(alu_tflops, 3), "peak": round(fma_peak, 3),
                "unit": "TFLOP/s", "frac": round(alu_tflops / fma_peak, 4), "traffic": ev.get("dram_bytes_per_launch"),
                "peak_source": f"measured in this run: mm_measure_fma_peak({w.dtype}), register-only FMA probe on all SMs",
                "peak_three_fresh_operands": round(fma_fresh3, 3), "frac_three_fresh_operands": round(alu_tflops / fma_fresh3, 4),
                "peak_nominal": round(nominal_fma, 2),
                "peak_nominal_derivation": "148 SMs x %d FMA lanes x 2 flops x 1.965 GHz" % (64 if w.dtype == "f64" else 128),
                "flops_per_cell_update": 2 * FMA_PER_CELL_UPDATE,
                "executed_inst_per_cell_update": ev.get("inst_per_cell_update"),
                "traffic_source": ev.get("source"), "fuse_T": fuse_t, "launches": n_launch,
                "avg_launch_ms": round(sub_ms / max(n_launch, 1), 4), "kernel_share_of_step": round(sub_ms / ms, 4),
                "note": "achieved = the method's 6 FMAs per cell-update (12 flops) x cell-updates of the timed mm_substep calls / "
                        "their CUDA-event time; the fused kernel moves one read + one write of the density per fuse_T substeps "
                        "and is bound by FMA issue, not HBM (roofline_hbm); an FMA pays for its fresh register operands at two "
                        "per cycle and scheduler (DESIGN.md section 8a): peak_three_fresh_operands = mm_measure_fma_rate(dtype, 3) "
                        "in this run is the rate of FMAs whose coefficient, value and accumulator all change, as this "
                        "stencil's do; about half of the executed instructions are the method's FMAs"}
    # (2) the HBM side: real DRAM rate of the fused pass, the algorithmic (T = 1 byte count) rate, the unfused kernel
    peak, peak_src = measured_peaks()
    alg_gbs = 2.0 * es * cell_updates / sub_s / 1e9                      # 2*sizeof(real) B per cell-update
    pass_gbs = 2.0 * es * g.cells * n_launch / sub_s / 1e9               # one fused pass: read once + write once
    hbm = {"bound": "hbm", "kernel": kname, "achieved": round(pass_gbs, 1), "peak": peak, "unit": "GB/s",
           "frac": round(pass_gbs / peak, 4), "traffic": ev.get("dram_bytes_per_launch"), "peak_source": peak_src,
           "frac_nominal_8tbs": round(pass_gbs / NOMINAL_HBM_GBS, 4),
           "effective_gbs": round(alg_gbs, 1), "effective_frac": round(alg_gbs / peak, 4),
           "effective_frac_nominal_8tbs": round(alg_gbs / NOMINAL_HBM_GBS, 4), "bytes_per_cell_update": 2 * es,
           "note": "achieved/frac = bytes the fused passes really move (one read + one write of the density per launch) / time; "
                   "effective_* = the algorithmic byte count of SURVEY 8(d) (2*sizeof(real) per cell-update, one substep per "
                   "pass) / time: above 1 because a launch fuses fuse_T substeps, not because memory is faster; t1_* = the "
                   "same kernel unfused, where both coincide -- north_star's >= 70 % of ~8 TB/s is stated on that point"}

    # ---- the same kernel unfused (T=1) for the T=1 roofline point (outside the timed region)
    if not args.no_t1 and fuse_t != 1 and not local_dt:
        mm.set_option(b.MM_OPT_FUSE_T, 1)
        mm.substep(3, w.dt)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        mm.substep(6, w.dt)
        e1.record(stream)
        torch.cuda.synchronize()
        t1 = 2.0 * es * g.cells * 6 / (e0.elapsed_time(e1) * 1e-3) / 1e9
        hbm.update({"t1_gbs": round(t1, 1), "t1_frac": round(t1 / peak, 4), "t1_frac_nominal_8tbs": round(t1 / NOMINAL_HBM_GBS, 4),
                    "t1_kernel": mm.kernel_name})
        mm.set_option(b.MM_OPT_FUSE_T, fuse_opt)

    extras = {}
    # ---- optional: NEXT-4 motor-force spreading of the current density (macro cadence; outside the timed region)
    if args.spread and full_protocol:
        psi = torch.rand(g.nc, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(7))
        F2 = torch.empty((g.nx, g.ny, 2), dtype=torch.float64, device=dev)
        mm.set_psi(psi)
        mm.spread_force(F2)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(3):
            mm.spread_force(F2)
        e1.record(stream)
        torch.cuda.synchronize()
        sms = e0.elapsed_time(e1) / 3
        extras["spread_force"] = {"ms_per_call": round(sms, 3), "density_read_gbs": round(g.cells * es / (sms * 1e-3) / 1e9, 1),
                                  "density_read_frac": round(g.cells * es / (sms * 1e-3) / 1e9 / peak, 4),
                                  "point_forces_per_call": g.nc * g.ns, "grid": [g.nx, g.ny]}

    # ---- optional: NEXT-2 free-motor coupling (macro cadence; outside the timed region; needs two buffers)
    if args.free and full_protocol:
        psi = torch.rand(g.nc, dtype=torch.float64, device=dev, generator=torch.Generator(device=dev).manual_seed(7))
        mm.set_psi(psi)
        Mf = torch.empty((g.nx, g.ny), dtype=torch.float64, device=dev)
        mm.update_free_motors(None, Mf)
        torch.cuda.synchronize()
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream)
        for _ in range(2):
            mm.update_free_motors(None, Mf)
        e1.record(stream)
        mm.substep(w.moments_every, w.dt)        # warm-up of the coupled-source kernels
        e1b = torch.cuda.Event(enable_timing=True)
        e1b.record(stream)
        mm.substep(2 * w.moments_every, w.dt)
        e2.record(stream)
        torch.cuda.synchronize()
        ums = e0.elapsed_time(e1) / 2
        extras["free_motors"] = {"update_ms_per_call": round(ums, 3),
                                 "density_read_gbs": round(g.cells * es / (ums * 1e-3) / 1e9, 1),
                                 "density_read_frac": round(g.cells * es / (ums * 1e-3) / 1e9 / peak, 4),
                                 "coupled_substep_kernel": mm.kernel_name,
                                 "coupled_substep_gcups": round(g.cells * 2 * w.moments_every / (e1b.elapsed_time(e2) * 1e-3) / 1e9, 2),
                                 "Mf_min": float(Mf.min().item()), "Mf_max": float(Mf.max().item())}
        mm.set_option(b.MM_OPT_FREE_COUPLING, 0)

    # ---- end to end: pinned host (U,V,Omega) in, moments out to pinned host, every step
    for _ in range(2 if full_protocol else 1):
        step(Up, Vp, Op, Fp, Tp)
    ms_e2e, _ = timed(steps, Up, Vp, Op, Fp, Tp)
    e2e = {"value": round(updates_per_step * steps / (ms_e2e * 1e-3) / 1e9, 2), "unit": UNIT,
           "h2d_bytes_per_step": int(3 * g.nc * es), "d2h_bytes_per_step": int(n_mom * 3 * g.nc * 8),
           "ms_per_step": round(ms_e2e / steps, 3),
           "note": "density is resident state (PAPER.md:133,143); per-step host traffic is (U,V,Omega) in, moments out"}
    return {"value": value, "ms": ms, "launches": launches, "clocks": clocks, "kname": kname, "e2e": e2e,
            "roofline": roofline, "roofline_hbm": hbm, "local_info": local_info, "extras": extras}


def make_context(w, args, dev, stream, log):
    import torch
    from paper_1908_04279_b200 import MM, binding as b
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    b0 = torch.empty(w.grid.cells, dtype=tdt, device=dev)
    b1 = None if args.single_buffer else torch.empty(w.grid.cells, dtype=tdt, device=dev)
    mm = MM(w.grid, w.params, w.dtype, b0, b1, stream=stream.cuda_stream)
    if args.fuse_t:
        mm.set_option(b.MM_OPT_FUSE_T, args.fuse_t)
    if args.kernel is not None:
        mm.set_option(b.MM_OPT_KERNEL, args.kernel)
    upload_inputs(mm, w, log=log)
    return mm, (b0, b1)


def run_cuda(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libmm has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def log(msg):
        if rank == 0:
            print(f"[bench] {msg}", file=sys.stderr, flush=True)

    free_b, _ = torch.cuda.mem_get_info()
    idx = pick_workload(args.config, free_b)
    w = with_scheme(rank_workload(mi.CONFIGS[idx], rank), args.scheme)
    if args.nx_mult > 1:   # a larger outer grid of the same structure (needs --single-buffer beyond 90 GB per buffer)
        g0 = w.grid
        w = mi.Workload(w.name + f"_nx{args.nx_mult}", mi.Grid(g0.nx * args.nx_mult, g0.ny, g0.ntheta, g0.ns, g0.nxi, g0.neta),
                        w.dtype, w.n_sub, w.moments_every, w.omega_max, w.seed, w.params)
    g, es = w.grid, ES[w.dtype]
    log(f"workload configs[{idx}] {w.name}: Nc={g.nc} cells={g.cells} dtype={w.dtype} n_sub={w.n_sub} "
        f"moments every {w.moments_every}; dt={w.dt:.6e}")

    stream = torch.cuda.current_stream()
    mm, bufs = make_context(w, args, dev, stream, log)
    r = measure(mm, w, idx, args, args.steps, args.warmup, dev, stream, world, log, full_protocol=True)
    mm.destroy()
    del mm, bufs
    torch.cuda.empty_cache()

    out = {"metric": METRIC, "value": round(r["value"], 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": round(r["ms"] / args.steps, 3), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": w.dtype, "data": "synthetic",
           "config": {"workload": f"configs[{idx}] {w.name}", "grid": [g.nx, g.ny, g.ntheta, g.ns, g.nxi, g.neta],
                      "cells_per_gpu": g.cells, "n_sub_per_step": w.n_sub, "moments_every": w.moments_every,
                      "dt": w.dt, "seed": w.seed, "parallelism": f"configs x{world} (no collective)",
                      "l2": "inputs larger than L2 (%s of %.1f GB)" % ("one density buffer, passes in place" if args.single_buffer else "two density buffers", g.cells * es / 1e9)},
           "clocks": r["clocks"], "e2e": r["e2e"], "gpu_launches": int(r["launches"]), "roofline": r["roofline"],
           "roofline_hbm": r["roofline_hbm"], "impl": "cuda"}
    out.update(r["extras"])
    if args.full:
        out["config"]["workload"] += "+full_step"
        out["full_step"] = {"per_macro_interval": "mm_update_free_motors, mm_substep (coupled source), mm_moments, mm_spread_force",
                            "note": "value still counts cell-updates of the substeps only; the roofline objects refer to the substep kernel"}
    if r["local_info"]:
        out["config"]["workload"] += "+local_dt"
        out["local_dt"] = r["local_info"]

    # ---- the other single-GPU workloads of BASELINE.json, a few steps each (driver-visible fp64 / medium-grid numbers)
    plain = not (args.full or args.local_dt or args.single_buffer or args.nx_mult > 1 or args.scheme != "euler")
    if rank == 0 and world == 1 and plain and not args.no_per_config and args.config is None:
        per = []
        for j in range(len(mi.CONFIGS)):
            if j == idx:
                continue
            wj = mi.CONFIGS[j]
            fb, _ = torch.cuda.mem_get_info()
            if 2 * wj.grid.cells * ES[wj.dtype] + (2 << 30) > fb:
                per.append({"workload": f"configs[{j}] {wj.name}", "skipped": "does not fit"})
                continue
            mmj, bj = make_context(wj, args, dev, stream, log)
            rj = measure(mmj, wj, j, args, 2, 1, dev, stream, 1, log, full_protocol=False)
            mmj.destroy()
            del mmj, bj
            torch.cuda.empty_cache()
            per.append({"workload": f"configs[{j}] {wj.name}", "dtype": wj.dtype, "value": round(rj["value"], 2), "unit": UNIT,
                        "steps": 2, "warmup": 1, "e2e": rj["e2e"]["value"], "kernel": rj["kname"],
                        "frac": rj["roofline"]["frac"], "fma_peak_tflops": rj["roofline"]["peak"],
                        "hbm_pass_frac": rj["roofline_hbm"]["frac"], "t1_frac": rj["roofline_hbm"].get("t1_frac"),
                        "t1_frac_nominal_8tbs": rj["roofline_hbm"].get("t1_frac_nominal_8tbs"), "clocks": rj["clocks"]})
        out["per_config"] = per
    if rank == 0 and world == 1 and not args.no_cpu and not args.local_dt:
        out["cpu_baseline"] = cpu_baseline(w, target_s=args.cpu_seconds, log=log)
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------- oracle arm
def oracle_sample(w, n_configs, reps=1):
    """Oracle (as it stands) on the first n_configs configurations of the workload: full step (n_sub substeps,
    moments at the cadence).  Returns seconds per step."""
    from oracle import mm_oracle as orc
    npdt = np.float64 if w.dtype == "f64" else np.float32
    st = mi.Stream(w.grid, w.params.R, w.seed, w.omega_max)
    U, V, Om = st.velocities(npdt)
    m = st.density(n_configs, npdt).astype(np.float64)
    st.close()
    U, V, Om = (np.asarray(x[:n_configs], np.float64) for x in (U, V, Om))
    times = []
    for _ in range(reps):
        t0 = time.perf_counter()
        for _k in range(w.n_sub // w.moments_every):
            m = orc.run(w.grid, w.params, U, V, Om, m, w.moments_every, w.dt)
            orc.moments(w.grid, w.params, m)
        times.append(time.perf_counter() - t0)
    return times


def cpu_baseline(w, target_s=15.0, log=None):
    from oracle import mm_oracle as orc
    cores = orc.threads()
    probe_n = 2 * cores
    t = oracle_sample(mi.Workload(w.name, w.grid, w.dtype, w.moments_every, w.moments_every, w.omega_max, w.seed,
                                  w.params), probe_n)[0]
    rate = probe_n * w.grid.inner * w.moments_every / t
    n = int(target_s * rate / (w.grid.inner * w.n_sub))
    n = max(cores, min(w.grid.nc, n // cores * cores))
    t = oracle_sample(w, n)[0]
    val = n * w.grid.inner * w.n_sub / t / 1e9
    if log:
        log(f"cpu_baseline: oracle on {n} configurations, {t:.1f} s, {val*1e3:.1f} M cell-updates/s on {cores} threads")
    out = {"value": round(val, 5), "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"first {n} of {w.grid.nc} configurations of the workload, all {w.n_sub} substeps + moments "
                     f"every {w.moments_every}; fp64; gcc -O2 -fopenmp over configurations", "seconds": round(t, 2)}
    # per-core figure (SURVEY.md 8(d) "additionally with 1 thread on configs[0]"): a child process, OMP_NUM_THREADS=1
    try:
        import subprocess
        code = ("import sys, json; sys.path.insert(0, %r); import bench, mm_inputs as mi; w = mi.CONFIGS[0]; n = 768; "
                "t = bench.oracle_sample(w, n)[0]; print(json.dumps([n, t]))" % ROOT)
        res = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300,
                             env={**os.environ, "OMP_NUM_THREADS": "1"})
        n1, t1 = json.loads(res.stdout.strip().splitlines()[-1])
        w0 = mi.CONFIGS[0]
        out["one_thread_configs0"] = {"value": round(n1 * w0.grid.inner * w0.n_sub / t1 / 1e9, 5), "unit": UNIT, "cores": 1,
                                      "sample": f"first {n1} of {w0.grid.nc} configurations of configs[0] fp64_tiny, all "
                                                f"{w0.n_sub} substeps + moments; OMP_NUM_THREADS=1", "seconds": round(t1, 2)}
    except Exception as e:   # the per-core figure is context: never fail the bench line over it
        out["one_thread_configs0"] = {"error": str(e)[:200]}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    free_b = None
    try:
        import torch
        if torch.cuda.is_available():
            free_b, _ = torch.cuda.mem_get_info()
    except Exception:
        pass
    idx = pick_workload(args.config, free_b)
    w = with_scheme(mi.CONFIGS[idx], args.scheme)
    g = w.grid
    from oracle import mm_oracle as orc
    cores = orc.threads()
    # size the per-step sample so that (warmup + steps) steps take about args.cpu_seconds * 4 in total
    probe_n = 2 * cores
    t = oracle_sample(mi.Workload(w.name, g, w.dtype, w.moments_every, w.moments_every, w.omega_max, w.seed, w.params),
                      probe_n)[0]
    rate = probe_n * g.inner * w.moments_every / t
    budget = 4.0 * args.cpu_seconds / max(1, args.steps + args.warmup)
    n = int(budget * rate / (g.inner * w.n_sub))
    n = max(cores, min(g.nc, n // cores * cores))
    times = oracle_sample(w, n, reps=args.warmup + args.steps)[args.warmup:]
    sec = sum(times)
    val = n * g.inner * w.n_sub * args.steps / sec / 1e9
    sample = (f"each step = first {n} of {g.nc} configurations of the workload, all {w.n_sub} substeps + moments every "
              f"{w.moments_every}; fp64 oracle, gcc -O2 -fopenmp over configurations")
    out = {"impl": "reference", "metric": METRIC, "value": round(val, 5), "unit": UNIT, "n_gpus": world,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(sec / args.steps * 1e3, 3),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"configs[{idx}] {w.name}", "grid": [g.nx, g.ny, g.ntheta, g.ns, g.nxi, g.neta],
                      "n_sub_per_step": w.n_sub, "moments_every": w.moments_every, "dt": w.dt, "seed": w.seed},
           "cpu_baseline": {"value": round(val, 5), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": round(val, 5), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=None, help="index into BASELINE.json configs (default: largest that fits)")
    ap.add_argument("--fuse-t", type=int, default=0, help="override MM_OPT_FUSE_T (0 = library default)")
    ap.add_argument("--kernel", type=int, default=None, help="override MM_OPT_KERNEL")
    ap.add_argument("--scheme", default="euler", choices=["euler", "rk2"],
                    help="euler = forward Euler + upwind (north_star, default); rk2 = RK2 + Superbee in s (NEXT-1)")
    ap.add_argument("--local-dt", action="store_true",
                    help="NEXT-3: advance each macro interval with mm_advance_local (per-configuration local steps)")
    ap.add_argument("--single-buffer", action="store_true",
                    help="create the context with ONE density buffer: every pass in place (MM_OPT_INPLACE), half the memory")
    ap.add_argument("--nx-mult", type=int, default=1, help="multiply the workload's Nx (a larger problem of the same structure)")
    ap.add_argument("--full", action="store_true",
                    help="time the whole microscale step: free-motor update + coupled substeps + moments + force spreading")
    ap.add_argument("--free", action="store_true",
                    help="NEXT-2: also time mm_update_free_motors and two substeps with the coupled source k_on M_f(r0)")
    ap.add_argument("--spread", action="store_true",
                    help="NEXT-4: also time mm_spread_force (motor-force spreading, Eq. 10) on the final density")
    ap.add_argument("--cfl", type=float, default=0.4, help="CFL number of --local-dt")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-t1", action="store_true", help="skip the unfused (T=1) roofline point")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of the other BASELINE workloads")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world and world == 1 and args.gpus > 1:
        raise SystemExit("launch N>1 with: python -m torch.distributed.run --nnodes=1 --nproc-per-node N "
                         "--master-addr 127.0.0.1 --master-port P bench.py --gpus N ...")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
