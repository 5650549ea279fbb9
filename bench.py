#!/usr/bin/env python
"""bench.py -- MLUPs and HBM-roofline fraction of the fused LBM step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

Workload at N = 1: BASELINE.json config 3 (configs[2]) -- D3Q19 Smagorinsky + HLBM, fp32, 384x192x128
urban channel -- the configuration the metric "MLUPs ... for D3Q19 Smagorinsky+HLBM" and the
north_star target are quoted on.  A "step" is one lattice time step = one pass of the whole hot path
 over all cells = one fused kernel launch (preceded by the wall-model pre-pass over the compact list of
WALLMODEL cells).  One step moves 1.46 GB, far more than the 126 MB L2, so no L2 flush is needed between steps.
Protocol: --repeats R (default 3) timed regions of exactly K steps, each from a fresh
lbm_init_equilibrium + W warm-up steps, CUDA events on the library's stream; the line reports the MEDIAN region
(all of them are listed in config.repeats_ms_per_step).  lbm_moments / lbm_totals (row A9) are timed separately
("moments" block) and are not part of MLUPs.
N > 1: the lattice is cut into z-slabs, one per GPU (one process per GPU), with one halo exchange per step over NCCL
send/recv (two in the HRR form): the 5 of 19 populations that cross each cut, lbm_set_halo / lbm_step_halo / lbm_halo_pack /
lbm_halo_unpack + paper_2506_21804_b200/slab.py.  Weak scaling by default: N copies of the workload's height stacked in z
(the same generator at (N nz, ny, nx)), value = all cell updates of the job / max time over ranks; --strong cuts the
workload's own lattice; --replicas (and the Vortex-Method workloads) run N independent replicas with no data-path collective.
--impl reference: the CPU oracle (oracle/), as it stands, timed on the host cores on a bounded sample.
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

import lbm_inputs as I  # noqa: E402

METRIC = "MLUPs"
UNIT = "MLUPs (1e6 non-SOLID lattice cell updates per second)"
WORKLOADS = {
    # name: (config number, shape (nz,ny,nx) or None for the config's own, dtype)
    "config3_urban_channel_384x192x128_f32": (3, None, "f32"),
    "config2_les_periodic_256_f32": (2, None, "f32"),
    "config4_d3q27_spheres_512_f32": (4, None, "f32"),
    "config3_urban_channel_384x192x128_f64": (3, None, "f64"),
    "config1_tgv_32_f64": (1, None, "f64"),
}
# config 5, the single-GPU capacity sweep: cubes 128^3 .. 896^3 (fp32) and 128^3 .. 640^3 (fp64)
for _n in (128, 256, 384, 512, 640, 768, 896):
    WORKLOADS["config5_urban_cube_%d_f32" % _n] = (5, (_n, _n, _n), "f32")
    if _n <= 640:
        WORKLOADS["config5_urban_cube_%d_f64" % _n] = (5, (_n, _n, _n), "f64")
# the paper's own collision (HRR, Eq. 6-11) on the config-3 / config-2 / config-4 inputs: sigma = 0.7 is this
# build's choice (the paper prints no value); wall-model cells take sigma = 0 (l.131)
HRR = dict(collision=1, sigma=0.7)
WORKLOADS["config3_urban_channel_384x192x128_f32_hrr"] = (3, None, "f32", HRR)
WORKLOADS["config3_urban_channel_384x192x128_f64_hrr"] = (3, None, "f64", HRR)
WORKLOADS["config2_les_periodic_256_f32_hrr"] = (2, None, "f32", HRR)
WORKLOADS["config4_d3q27_spheres_512_f32_hrr"] = (4, None, "f32", HRR)
WORKLOADS["config5_urban_cube_512_f32_hrr"] = (5, (512, 512, 512), "f32", HRR)
# the same collision with the FD strain of the previous level's u^ (collision = 2, reading G41): one pass per step
HRRLAG = dict(collision=2, sigma=0.7)
WORKLOADS["config3_urban_channel_384x192x128_f32_hrrlag"] = (3, None, "f32", HRRLAG)
WORKLOADS["config3_urban_channel_384x192x128_f64_hrrlag"] = (3, None, "f64", HRRLAG)
WORKLOADS["config2_les_periodic_256_f32_hrrlag"] = (2, None, "f32", HRRLAG)
WORKLOADS["config4_d3q27_spheres_512_f32_hrrlag"] = (4, None, "f32", HRRLAG)
WORKLOADS["config5_urban_cube_512_f32_hrrlag"] = (5, (512, 512, 512), "f32", HRRLAG)
# lid-driven cavity, the paper's own scaling benchmark (fp32): closed box, moving lid
for _n in (256, 512, 640):
    WORKLOADS["cavity_%d_f32" % _n] = (6, (_n, _n, _n), "f32")
WORKLOADS["cavity_512_f32_hrr"] = (6, (512, 512, 512), "f32", HRR)
WORKLOADS["cavity_512_f32_hrrlag"] = (6, (512, 512, 512), "f32", HRRLAG)
# Vortex Method inlet (Eq. 18-21) on the config-3 channel: power-law mean profile, 256 seeded vortices of size 6 cells,
# intensity 0.15; "_hrr_vm" = the paper's urban set-up as far as this build has it (HRR + Smagorinsky + HLBM + wall model + VM)
VM = dict(n_vortices=256, sigma_v=6.0, intensity=0.15)
WORKLOADS["config3_urban_channel_384x192x128_f32_vm"] = (3, None, "f32", {}, VM)
WORKLOADS["config3_urban_channel_384x192x128_f32_hrr_vm"] = (3, None, "f32", HRR, VM)
WORKLOADS["config3_urban_channel_384x192x128_f32_hrrlag_vm"] = (3, None, "f32", HRRLAG, VM)
# the urban channel in the paper's own boundary set (l.255: fixed-pressure outlet + fringe zone, full-slip outer walls, wall-modelled
# floor) with the VM inlet; "_hrr_vm" is the paper's HHRRLBM-LES urban set-up as far as the paper defines it
WORKLOADS["paperbc_urban_channel_384x192x128_f32_vm"] = (7, (128, 192, 384), "f32", {}, VM)
WORKLOADS["paperbc_urban_channel_384x192x128_f32_hrr_vm"] = (7, (128, 192, 384), "f32", HRR, VM)
WORKLOADS["paperbc_urban_channel_384x192x128_f32_hrrlag_vm"] = (7, (128, 192, 384), "f32", HRRLAG, VM)
# moving porous bodies (Eq. 12 with u^B != 0): the trees of config 3 (0 < d < 1, 5 % of the cells) sway with a seeded
# solid velocity field (lbm_inputs.body_velocity), set once through lbm_set_body_velocity
BODY = dict(amp=0.02)
WORKLOADS["config3_urban_channel_384x192x128_f32_body"] = (3, None, "f32", {}, None, BODY)
WORKLOADS["config3_urban_channel_384x192x128_f32_hrr_body"] = (3, None, "f32", HRR, None, BODY)
# the paper's boundary set with the wall model on the building faces too (config 8; SURVEY 8(f)-2 "wall model on building faces")
WORKLOADS["paperbc_wmfaces_urban_channel_384x192x128_f32_vm"] = (8, (128, 192, 384), "f32", {}, VM)
WORKLOADS["paperbc_wmfaces_urban_channel_384x192x128_f32_hrr_vm"] = (8, (128, 192, 384), "f32", HRR, VM)
WORKLOADS["paperbc_wmfaces_urban_channel_384x192x128_f32_hrrlag_vm"] = (8, (128, 192, 384), "f32", HRRLAG, VM)
# propagation bake-off: the fully periodic LES box of config 2 on two lattices (pull) and in place (AA pattern,
# option "inplace"); at 768^3 fp64 one population set is 68.9 GB
INPLACE = dict(inplace=1)
WORKLOADS["config2_les_periodic_256_f32_inplace"] = (2, None, "f32", {}, None, None, INPLACE)
WORKLOADS["config4_d3q27_spheres_512_f32_inplace"] = (4, None, "f32", {}, None, None, INPLACE)
for _n, _t in ((512, "f32"), (768, "f64")):
    WORKLOADS["config2_les_periodic_%d_%s" % (_n, _t)] = (2, (_n, _n, _n), _t)
    WORKLOADS["config2_les_periodic_%d_%s_inplace" % (_n, _t)] = (2, (_n, _n, _n), _t, {}, None, None, INPLACE)
DEFAULT_WORKLOAD = "config3_urban_channel_384x192x128_f32"


def workload(name):
    """-> (config number, shape or None, dtype, extra lbm_params)"""
    w = WORKLOADS[name]
    return (w[0], w[1], w[2], dict(w[3]) if len(w) > 3 else {})


def workload_vm(name, shape):
    """Vortex Method inlet inputs of the workload (lbm_inputs.vm_inlet) or None"""
    w = WORKLOADS[name]
    if len(w) < 5 or w[4] is None:
        return None
    return I.vm_inlet(shape, 1300 + w[0], **w[4])


def workload_body(name, cfg):
    """solid velocity field u^B of the workload (lbm_inputs.body_velocity) or None"""
    w = WORKLOADS[name]
    if len(w) < 6 or w[5] is None:
        return None
    return I.body_velocity(cfg, 1400 + w[0], **w[5])


def oracle_steps(O, f, cfg, vm, state, nsteps, nthreads):
    """the oracle's step loop, with the VM inlet when the workload has one (state = the previous inflow, carried along)"""
    kw = dict(d=cfg["d"], flags=cfg["flags"], nsteps=nsteps, nthreads=nthreads, **cfg["params"])
    if cfg.get("u_body") is not None:
        kw["u_body"] = cfg["u_body"]
    if vm is None:
        return O.step(f, **kw), None
    return O.step_vm(f, vm["u_mean"], vm["u_mean"] if state is None else state, vm["pos"], vm["sign"], vm["sigma_v"],
                     vm["intensity"], **kw)


def make_cfg(number, shape, extra):
    cfg = I.make_config(number, shape=shape) if number != 1 else I.make_config(1)
    cfg["params"] = dict(cfg["params"], **extra)
    return cfg


def make_cfg_named(name, number, shape, extra):
    cfg = make_cfg(number, shape, extra)
    cfg["u_body"] = workload_body(name, cfg)
    return cfg


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/ncu_traffic.csv)."""
    import csv
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(p):
        return None
    for row in csv.DictReader(open(p)):
        if row["workload"] == workload:
            return int(row["dram_read_bytes_per_launch"]) + int(row["dram_write_bytes_per_launch"])
    return None


def algorithmic_bytes_per_step(cfg, dtype, n_solid):
    """2*Q*sizeof(T) + sizeof(T) (porosity, when use_hlbm) + 1 (flag) per non-SOLID cell,
    1 byte per SOLID cell."""
    sz = 4 if dtype == "f32" else 8
    N = int(np.prod(cfg["shape"]))
    per_cell = 2 * cfg["Q"] * sz + (sz if cfg["params"].get("use_hlbm") else 0) + 1
    return (N - n_solid) * per_cell + n_solid * 1, per_cell


def max_over_ranks(x, world, device="cuda"):
    """Replicas-only multi-GPU: the job time is the max over ranks (all_reduce MAX; a no-op for one rank)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    if dist.get_backend() == "gloo":
        device = "cpu"
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_mlups(world, units_per_rank, steps, seconds):
    """Whole-job throughput: every rank processed units_per_rank * steps cell updates in `seconds` (max over ranks)."""
    return world * units_per_rank * steps / seconds / 1e6


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_evt = index, [], set(), None, threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.005)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def cpu_oracle_time(cfg_number, sample_shape, nsteps, nthreads, extra, name):
    """Time the oracle, as it stands, on a bounded sample of the workload."""
    from oracle import oracle as O
    cfg = make_cfg_named(name, cfg_number, sample_shape, extra)
    vm = workload_vm(name, cfg["shape"])
    f = O.init_equilibrium(cfg["Q"], cfg["rho"], cfg["u"])
    nonsolid = f[0].size if cfg["flags"] is None else int((~I.is_wall(cfg["flags"])).sum())
    oracle_steps(O, f, cfg, vm, None, 1, nthreads)                                              # warm-up
    t0 = time.perf_counter()
    oracle_steps(O, f, cfg, vm, None, nsteps, nthreads)
    dt = time.perf_counter() - t0
    return nonsolid * nsteps / dt / 1e6, dt, cfg["shape"]


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import oracle as O
    number, shape, dtype, extra = workload(args.workload)
    cores = O.max_threads()
    if world > 1:
        # torchrun exports OMP_NUM_THREADS=1 to every rank; rank 0 is the only one that works here, so it takes the host cores it may
        # run on (the oracle takes its thread count as an argument)
        cores = max(cores, len(os.sched_getaffinity(0)))
    total = max(args.steps + args.warmup, 1)
    # bounded sample: a reduced instance of the same generator, sized for roughly a minute in total
    cells_budget = max(int(60.0 * 1.0e6 / total), 4096)
    if number == 1:
        sample = (32, 32, 32)
    else:
        base = {2: (256, 256, 256), 3: (128, 192, 384), 4: (512, 512, 512), 5: shape, 6: shape, 7: shape, 8: shape}[number]
        scale = min(1.0, (cells_budget / float(np.prod(base))) ** (1.0 / 3.0))
        sample = tuple(max(16, int(round(b * scale / 8)) * 8) for b in base)
    cfg = make_cfg_named(args.workload, number, sample, extra)
    f = O.init_equilibrium(cfg["Q"], cfg["rho"], cfg["u"])
    nonsolid = f[0].size if cfg["flags"] is None else int((~I.is_wall(cfg["flags"])).sum())
    vm = workload_vm(args.workload, cfg["shape"])
    f, st = oracle_steps(O, f, cfg, vm, None, args.warmup, cores)
    t0 = time.perf_counter()
    f, st = oracle_steps(O, f, cfg, vm, st, args.steps, cores)
    dt = time.perf_counter() - t0
    value = nonsolid * args.steps / dt / 1e6
    sample_txt = "oracle (fp64, %d OpenMP threads) on the workload generator at (nz,ny,nx)=%s, %d steps" % (
        cores, str(tuple(sample)), args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / max(args.steps, 1) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "sample_shape_nz_ny_nx": list(sample)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_txt},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--repeats", type=int, default=3, help="timed regions of K steps each, every one from a fresh state; the median is reported")
    ap.add_argument("--replicas", action="store_true", help="N > 1: independent replicas instead of the z-slab decomposition")
    ap.add_argument("--strong", action="store_true", help="N > 1: cut the workload's own lattice N ways (strong scaling) instead of stacking N of them in z")
    ap.add_argument("--no-moments", action="store_true", help="skip the separate timing of lbm_moments / lbm_totals (A9)")
    ap.add_argument("--option", action="append", default=[], help="library option key=value (tuning)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if args.steps is None:
            args.steps = 10
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    import paper_2506_21804_b200 as P

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    # LBM_BENCH_ONE_GPU=1: a dry run of the N > 1 path on ONE GPU (all ranks on cuda:0, halos exchanged through gloo and the host;
    # nothing in a kernel ever waits for another rank).  It checks the decomposition end to end; its numbers are not a measurement.
    one_gpu = os.environ.get("LBM_BENCH_ONE_GPU") == "1"
    if one_gpu:
        local_rank = 0
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if one_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    number, shape, dtype, extra = workload(args.workload)
    # N > 1: the lattice is cut into z-slabs, one per GPU, with a halo exchange per step.  Weak scaling
    # (default): N copies of the workload's height stacked in z -- the same generator at (N nz, ny, nx) -- so every GPU keeps the
    # workload's own cell count; --strong cuts the workload's own lattice.  Workloads with the Vortex Method inlet (it needs the
    # whole inflow plane) and config 1 run as independent replicas.
    decomposed = world > 1 and not args.replicas and number != 1 and workload_vm(args.workload, (8, 8, 8)) is None
    if decomposed and not args.strong:
        base = shape or make_cfg(number, None, {})["shape"]
        shape = (base[0] * world, base[1], base[2])
    cfg = make_cfg_named(args.workload, number, shape, extra)
    hrr = cfg["params"].get("collision", 0) >= 1
    if args.steps is None:
        args.steps = cfg["steps"]
    Q = cfg["Q"]
    tdt = torch.float32 if dtype == "f32" else torch.float64
    npdt = np.float32 if dtype == "f32" else np.float64
    par = P.LbmParams(**cfg["params"])
    stream = torch.cuda.current_stream()
    part = None
    n_wall_global = 0 if cfg["flags"] is None else int(I.is_wall(cfg["flags"]).sum())
    cells_global = int(np.prod(cfg["shape"]))
    if decomposed:
        from paper_2506_21804_b200 import slab as S
        gnz, ny, nx = cfg["shape"]
        part = S.SlabLBM(Q, nx, ny, gnz, dtype, rank, world, S.z_is_closed(cfg["flags"]), stream=stream.cuda_stream)
        sim = part.sim
        sl = part.slab
        for key, axis in (("rho", 0), ("u", 1), ("d", 0), ("flags", 0), ("u_body", 1)):
            if cfg.get(key) is not None:
                cfg[key] = sl.take(cfg[key], axis=axis)           # this rank's slices, ghost slices included
        nz = sl.nz_local
    else:
        nz, ny, nx = cfg["shape"]
        sim = P.LBM(Q, nx, ny, nz, dtype, stream=stream.cuda_stream)
    N = nx * ny * nz
    wl = WORKLOADS[args.workload]
    for k, v in (wl[6] if len(wl) > 6 else {}).items():
        sim.set_option(k, v)
    for kv in args.option:
        k, v = kv.split("=")
        sim.set_option(k, int(v))

    def do_steps(n):
        if part is not None:
            part.step(n, par)
        else:
            sim.step(n, par)

    # inputs resident in HBM before the timed region
    rho_d = torch.from_numpy(cfg["rho"].astype(npdt)).cuda()
    u_d = torch.from_numpy(cfg["u"].astype(npdt)).cuda()
    d_d = None if cfg["d"] is None else torch.from_numpy(cfg["d"].astype(npdt)).cuda()
    fl_d = None if cfg["flags"] is None else torch.from_numpy(cfg["flags"]).cuda()
    sim.set_geometry(d_d, fl_d)
    if part is not None:
        part.init_equilibrium(rho_d, u_d)                     # + lbm_set_halo
    else:
        sim.init_equilibrium(rho_d, u_d)
    if cfg.get("u_body") is not None:
        sim.set_body_velocity(torch.from_numpy(cfg["u_body"].astype(npdt)).cuda())
    vm = workload_vm(args.workload, cfg["shape"])
    if vm is not None:
        sim.set_inflow(torch.from_numpy(vm["u_mean"].astype(npdt)).cuda())
        sim.set_vortices(vm["pos"], vm["sign"], vm["sigma_v"], vm["intensity"])
    if decomposed:
        n_solid = n_wall_global                               # job-wide counts (every rank generated the global geometry)
        n_fluid = (cells_global - n_wall_global) / world      # per rank on average: job value = world * n_fluid * steps / time
    else:
        n_solid = sim.query("solid_cells")
        n_fluid = N - n_solid

    def job_totals():
        t = np.array(sim.totals())
        if decomposed:
            tt = torch.tensor(t, device="cpu" if dist.get_backend() == "gloo" else "cuda", dtype=torch.float64)
            dist.all_reduce(tt)
            t = tt.cpu().numpy()
        return t

    tot0 = job_totals()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: R regions of exactly K steps, each from a fresh state + W warm-up steps -----------
    sampler = ClockSampler(local_rank)
    sampler.start()
    region_ms, launches = [], 0
    for rep in range(max(args.repeats, 1)):
        if rep > 0:
            (part or sim).init_equilibrium(rho_d, u_d)        # fresh S_0 (also resets the inflow history of the VM inlet)
        do_steps(args.warmup)
        barrier()
        l0 = sim.query("launches")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        do_steps(args.steps)
        e1.record(stream)
        barrier()
        launches = sim.query("launches") - l0
        region_ms.append(max_over_ranks(e0.elapsed_time(e1), world))
    clocks = sampler.stop()
    ms = float(np.median(region_ms))
    tot1 = job_totals()
    finite = bool(np.isfinite(tot1).all())
    value = job_mlups(world, n_fluid, args.steps, ms * 1e-3)
    step_bytes, per_cell = algorithmic_bytes_per_step(cfg, dtype, n_solid)
    if decomposed:
        step_bytes //= world                                  # per GPU (the roofline figures are per GPU)
    peak, peak_src = measured_peak()
    # BGK form: one launch over the lattice = one step.  HRR form: a step is two launches over the lattice (u^ pass + fused step);
    # the figure is then algorithmic bytes per STEP / time per step, i.e. it charges the u^ pass to the step kernel
    achieved = step_bytes / (ms * 1e-3 / max(args.steps, 1)) / 1e9    # GB/s

    # ---- A9, timed separately (not part of MLUPs): lbm_moments / lbm_totals on the stepped state (post-collision storage:
    # the pull happens in registers).  Algorithmic bytes: (Q + 4) sizeof(T) N resp. Q sizeof(T) N (+ 1 class byte per cell)
    moments = None
    if not args.no_moments:
        sz = 4 if dtype == "f32" else 8
        rho_o = torch.empty((nz, ny, nx), dtype=tdt, device="cuda")
        u_o = torch.empty((3, nz, ny, nx), dtype=tdt, device="cuda")

        def timed(fn, n=7):
            fn()
            ts = []
            for _ in range(n):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                fn()
                b.record(stream)
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            return max_over_ranks(float(np.median(ts)), world)

        lm0 = sim.query("launches")
        t_mom = timed(lambda: sim.moments(rho_o, u_o))
        lm1 = sim.query("launches")
        tot_o = torch.empty(5, dtype=torch.float64, device="cuda")
        t_tot = timed(lambda: sim.totals(tot_o))
        lm2 = sim.query("launches")
        b_mom = (Q + 4) * sz * n_fluid + N
        b_tot = Q * sz * n_fluid + N
        moments = {"lbm_moments": {"ms": t_mom, "algorithmic_bytes": b_mom, "achieved_gbs": b_mom / (t_mom * 1e-3) / 1e9,
                                   "frac": b_mom / (t_mom * 1e-3) / 1e9 / peak, "launches_per_call": (lm1 - lm0) / 8.0},
                   "lbm_totals": {"ms": t_tot, "algorithmic_bytes": b_tot, "achieved_gbs": b_tot / (t_tot * 1e-3) / 1e9,
                                  "frac": b_tot / (t_tot * 1e-3) / 1e9 / peak, "launches_per_call": (lm2 - lm1) / 8.0,
                                  "note": "result into a device buffer (asynchronous; a host buffer adds the copy and a stream synchronisation)"},
                   "what": "median of 7 calls on the stepped state, CUDA events; device outputs rho[N], u[3][N]; not part of MLUPs"}
        del rho_o, u_o

    # ---- end to end through the C ABI with HOST buffers ------------------------------------------
    # The workload's inputs are the macroscopic fields the generator writes (rho, u, porosity, flags): the timed region copies them
    # from pinned host memory (lbm_set_geometry + lbm_init_equilibrium build the state on the device), runs the K steps and reads
    # rho, u back to the host.  "from_populations" times the heavier entry as well: the full population set handed in from the host.
    e2e = None
    if not args.no_e2e:
        h_d = None if cfg["d"] is None else torch.from_numpy(cfg["d"].astype(npdt)).pin_memory()
        h_fl = None if cfg["flags"] is None else torch.from_numpy(cfg["flags"]).pin_memory()
        h_rho_in = torch.from_numpy(cfg["rho"].astype(npdt)).pin_memory()
        h_u_in = torch.from_numpy(cfg["u"].astype(npdt)).pin_memory()
        h_rho = torch.empty((nz, ny, nx), dtype=tdt).pin_memory()
        h_u = torch.empty((3, nz, ny, nx), dtype=tdt).pin_memory()
        sim.moments(h_rho, h_u)                        # warms the staging buffer
        size = lambda t: 0 if t is None else t.numel() * t.element_size()
        d2h = size(h_rho) + size(h_u)

        def timed_e2e(load):
            barrier()
            t0 = time.perf_counter()
            load()
            do_steps(args.steps)
            sim.moments(h_rho, h_u)                    # D2H: rho, u
            sim.synchronize()
            return max_over_ranks(time.perf_counter() - t0, world)

        def load_fields():
            sim.set_geometry(h_d, h_fl)                # H2D: porosity + flags
            (part or sim).init_equilibrium(h_rho_in, h_u_in)    # H2D: rho, u

        dt = timed_e2e(load_fields)
        h2d = size(h_d) + size(h_fl) + size(h_rho_in) + size(h_u_in)
        e2e = {"value": job_mlups(world, n_fluid, args.steps, dt), "unit": UNIT,
               "h2d_bytes_per_step": h2d / args.steps, "d2h_bytes_per_step": d2h / args.steps,
               "what": "lbm_set_geometry(host porosity, flags) + lbm_init_equilibrium(host rho, u) + lbm_step(K) + lbm_moments(host rho, u), wall clock"}
        if Q * N * (4 if dtype == "f32" else 8) < 8e9:          # (a pinned copy of the populations: bounded)
            h_f = torch.empty((Q, nz, ny, nx), dtype=tdt).pin_memory()
            (part or sim).init_equilibrium(rho_d, u_d)
            sim.get_populations(h_f)                   # host copy of S_0 (not timed)
            dt2 = timed_e2e(lambda: sim.set_fields(h_f, h_d, h_fl))     # H2D: populations + porosity + flags
            e2e["from_populations"] = {"value": job_mlups(world, n_fluid, args.steps, dt2),
                                       "h2d_bytes_per_step": (size(h_f) + size(h_d) + size(h_fl)) / args.steps,
                                       "what": "lbm_set_fields(host populations, porosity, flags) + lbm_step(K) + lbm_moments(host rho, u)"}

    # ---- CPU oracle beside it (rank 0, N = 1 only; bounded sample) -------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        cores = O.max_threads()
        if number == 1:
            sample_shape, ns = None, 2000
        else:
            base = np.array(cfg["shape"], dtype=float)
            scale = min(1.0, (1.5e6 / base.prod()) ** (1.0 / 3.0))
            sample_shape = tuple(max(16, int(round(b * scale / 8)) * 8) for b in base)
            ns = 100   # ~1.5e8 cell updates: about 10 s of host work at the oracle's ~15 MLUPs
        v, dt_cpu, shp = cpu_oracle_time(number, sample_shape, ns, cores, extra, args.workload)
        ns1 = max(ns // 10, 1)                                 # the same sample on ONE thread, a tenth of the steps
        v1, dt1, _ = cpu_oracle_time(number, sample_shape, ns1, 1, extra, args.workload)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "fp64 oracle, %d OpenMP threads, workload generator at (nz,ny,nx)=%s, %d steps after 1 warm-up, %.1f s"
                         % (cores, str(tuple(shp)), ns, dt_cpu),
               "single_thread": {"value": v1, "unit": UNIT, "cores": 1,
                                 "sample": "the same sample, 1 thread, %d steps after 1 warm-up, %.1f s" % (ns1, dt1)}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if (decomposed and args.strong) else "weak", "vs_baseline": None,
            "dtype": dtype, "data": "synthetic",
            "config": {"workload": args.workload, "lattice": "D3Q%d" % Q, "nx": nx, "ny": ny, "nz": nz, "cells": N,
                       "solid_cells": n_solid, "masked_cells": sim.query("masked_cells"), "params": cfg["params"],
                       "l2": "inputs larger than L2 (%.2f GB per step)" % (step_bytes / 1e9),
                       "mlups_all_cells": (cells_global if decomposed else world * N) * args.steps / (ms * 1e-3) / 1e6,
                       "parallelism": ("z-slabs, one per GPU, halo exchange per step over %s (%s scaling): global lattice %s"
                                       % ("gloo through the host, ALL RANKS ON ONE GPU: a dry run, not a measurement" if one_gpu else "NCCL send/recv",
                                          "strong" if args.strong else "weak", "x".join(str(v) for v in cfg["shape"][::-1]))) if decomposed
                                      else ("replicas only" if world > 1 else "single GPU"),
                       "finite": finite, "mass_drift_rel": (tot1[0] - tot0[0]) / tot0[0],
                       "repeats_ms_per_step": [t / args.steps for t in region_ms],
                       "protocol": "median of %d timed regions of %d steps, each from a fresh lbm_init_equilibrium + %d warm-up steps" % (len(region_ms), args.steps, args.warmup),
                       "bytes_per_update": per_cell},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": ncu_traffic(args.workload), "traffic_source": "profiles/ncu_traffic.csv (ncu --set full capture of this workload, DRAM read + write bytes per launch)",
                         "peak_source": peak_src, "frac_of_8000_datasheet": achieved / 8000.0,
                         "algorithmic_bytes_per_launch": step_bytes, "kernel": "lbm::k_step_vec<%d,%s,MODE_STREAM_COLLIDE,%s>" % (Q, "float" if dtype == "f32" else "double", "COLL_HRR" if hrr else "COLL_BGK"),
                         "launches_per_step": launches / max(args.steps, 1)},
            "moments": moments, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    sim.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
