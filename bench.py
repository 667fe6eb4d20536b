#!/usr/bin/env python
"""bench.py -- headline measurement: fp64 cell-updates/s per RK2 step at 256^3 (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3|4|2|0]

A "step" is one pass of the whole hot path (ghost fill, stage 1, ghost fill, stage 2 with fused
CFL reduction, device-side dt) over the whole grid.  `value` is timed with CUDA events on the
library's stream with the state already resident in HBM (hydro_run_steps, CUDA-graph replay); per-kernel
times for the roofline come from a second pass of the same steps with every launch bracketed by
events; `e2e` is the same step
through the C-ABI with HOST buffers: every timed step copies the state host->device
(hydro_set_state from pinned memory), runs hydro_cfl_dt + hydro_step, and copies it back
(hydro_get_state) -- the transfer pattern of the paper's Algorithm 2.
One JSON line on stdout (rank 0).  N > 1: independent replicas, one per GPU (DESIGN.md section 9:
"replicas only"; the path has no exchange step on one domain), no data-path collective.
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

METRIC = "fp64 cell-updates/sec per RK2 step at 256^3; achieved HBM GB/s vs B200 peak"
UNIT = "cell-updates/s"
# algorithmic HBM bytes per cell: stage 1 reads U0 and writes U1 (2 x 40 B),
# stage 2 reads U1 and U0 and writes U(n+1) (3 x 40 B)
BYTES_STAGE = {1: 80.0, 2: 120.0}
# algorithmic fp64-pipe instructions per cell per stage (primitives 13, 15 slopes
# x 9, 3 HLL fluxes x 62, update 30 / 40, fused signal speed 0 / 31; each slope and face once, no halo)
# and the measured fp64 pipe peak: 63 lanes/clk/SM x 148 SM at clocks.max.sm (DFMA/DADD/DMUL microbenchmark)
FP64_INSTR_STAGE = {1: 364.0, 2: 405.0}
# shared-memory crossbar: 128 B/clk/SM; bytes the threads and the TMA unit move through it per cell and
# stage (86 eight-byte accesses per thread and plane + the 36 x 20 x 40 B box)
SMEM_BYTES_CELL_STAGE = 86 * 8.0 + 36 * 20 * 40.0 / 512
FP64_LANES_PER_SM, N_SM = 63, 148


def max_over_ranks(x, world, device):
    """MAX-reduce a host float over the ranks of the default process group (N > 1)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def csrc_sha256():
    """Hash of the CUDA sources the library is built from: keys the committed ncu capture."""
    import hashlib
    d = os.path.join(ROOT, "paper_1812_07977_b200", "csrc")
    hsh = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            hsh.update(f.encode())
            hsh.update(open(os.path.join(d, f), "rb").read())
    return hsh.hexdigest()[:16]


def load_traffic(config):
    """roofline.traffic comes from a committed `ncu --set full` capture (a bench run is never taken
    under a profiler).  profiles/traffic.txt names the sources it was captured from (csrc_sha256);
    a capture of other sources is refused, so the number cannot go stale silently."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    out = {"dram": None, "fp64": None, "source": "no committed capture (profiles/traffic.txt absent)"}
    if not os.path.exists(p):
        return out
    kv = {}
    for ln in open(p):
        f = ln.split()
        if len(f) == 2 and not ln.startswith("#"):
            kv[f[0]] = f[1]
    have, want = kv.get("csrc_sha256"), csrc_sha256()
    if have != want:
        out["source"] = f"stale capture refused: profiles/traffic.txt is of csrc {have}, library is {want}"
        return out
    if f"config{config}" in kv:
        out["dram"] = float(kv[f"config{config}"])
    if f"config{config}_fp64_executed" in kv:
        out["fp64"] = float(kv[f"config{config}_fp64_executed"])
    out["source"] = (f"committed ncu --set full capture of csrc {have} "
                     f"({kv.get('capture', 'profiles/')}), per stage-pair launch")
    return out


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0=None, t1=None):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.08)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for (t, r) in self.rows if (t0 is None or t >= t0) and (t1 is None or t <= t1)]
        if not rows:
            rows = [r for _, r in self.rows]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)),
                "power_w_max": float(max(pw)), "samples": len(sm), "reasons": sorted(reasons)}


def workload(idx):
    from paper_1812_07977_b200 import inputs
    cfg = inputs.config(idx)
    return cfg


def cfg_dict(cfg, extra=None):
    d = {"workload": f"BASELINE.json configs[{cfg.index}]: {cfg.name}", "grid": list(cfg.shape),
         "gamma": cfg.gamma, "cfl": cfg.cfl, "bc": list(cfg.bc), "limiter_theta": cfg.theta,
         "l2": "state (2 padded buffers) larger than L2; no flush needed"}
    if extra:
        d.update(extra)
    return d


# ------------------------------------------------------------------------------------------
# oracle legs (the only places bench.py may execute oracle/)
# ------------------------------------------------------------------------------------------

def oracle_slab_state(cfg, nzs):
    """Bounded sample of the workload: the central nzs z-planes of the config's initial state."""
    U = cfg.state()
    nz = cfg.shape[2]
    z0 = (nz - nzs) // 2
    return np.ascontiguousarray(U[:, z0:z0 + nzs])


def time_oracle(cfg, steps, warmup, nzs):
    import oracle
    U = oracle_slab_state(cfg, nzs)
    nx, ny = cfg.shape[0], cfg.shape[1]
    o = oracle.OracleHydro(nx, ny, nzs, cfg.gamma, cfg.dx, cfg.bc)
    o.set_cfl(cfg.cfl)
    o.set_state(U)
    for _ in range(warmup):
        o.step(o.cfl_dt())
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(o.cfl_dt())
    el = time.perf_counter() - t0
    cells = nx * ny * nzs
    return cells * steps / el, el, oracle.get_threads(), cells


def cpu_baseline(cfg, budget_s=20.0):
    """Oracle as it stands on the host cores, on a bounded sample (~10-30 s of CPU work)."""
    nz = cfg.shape[2]
    rate, _, cores, _ = time_oracle(cfg, 1, 0, min(nz, 32))      # calibrate (also warms up)
    plane = cfg.shape[0] * cfg.shape[1]
    steps = 2
    nzs = int(max(8, min(nz, budget_s * rate / (plane * steps))))
    if nzs == nz:                                                # whole grid fits: add steps
        steps = int(max(2, min(50, budget_s * rate / (plane * nz))))
    rate, el, cores, cells = time_oracle(cfg, steps, 0, nzs)
    return {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{cfg.name}: central {cfg.shape[0]}x{cfg.shape[1]}x{nzs} slab, {steps} RK2 "
                      f"steps, {el:.1f} s wall"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload(args.config)
    nz = cfg.shape[2]
    rate, _, cores, _ = time_oracle(cfg, 1, 0, min(nz, 16))
    plane = cfg.shape[0] * cfg.shape[1]
    total = args.steps + args.warmup
    nzs = int(max(8, min(nz, 120.0 * rate / (plane * total))))      # whole run ~2 min
    rate, el, cores, cells = time_oracle(cfg, args.steps, args.warmup, nzs)
    sample = (f"{cfg.name}: central {cfg.shape[0]}x{cfg.shape[1]}x{nzs} slab per step, "
              f"{args.steps} timed RK2 steps")
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": cfg_dict(cfg, {"sample_cells_per_step": cells}),
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------

def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1812_07977_b200.binding import Hydro, load_library

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    # HYDRO_BENCH_BACKEND=gloo lets the N > 1 path (rendezvous, barriers, max-over-ranks timing) be
    # exercised on a box with fewer GPUs than ranks: the replicas then share devices (they only meet
    # at host-side barriers, no kernel waits on another rank)
    backend = os.environ.get("HYDRO_BENCH_BACKEND", "nccl")
    local = local % torch.cuda.device_count() if backend != "nccl" else local
    torch.cuda.set_device(local)
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    red_dev = "cuda" if backend == "nccl" else "cpu"

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = workload(args.config)
    L = load_library(False)
    traffic = load_traffic(args.config)
    hbm_peak, peak_src, sm_max = load_peaks()
    cells = cfg.cells

    h = Hydro(*cfg.shape, cfg.gamma, cfg.dx, cfg.bc)
    h.set_cfl(cfg.cfl)
    if args.variant is not None:
        h.set_kernel_variant(args.variant)
    if args.tile_rows or args.planes_per_chunk:
        h.set_tiling(args.tile_rows, args.planes_per_chunk)
    tiling = h.get_tiling()
    U0 = torch.from_numpy(cfg.state()).pin_memory()        # pinned host copy of the input
    Ud = U0.cuda(non_blocking=True)
    torch.cuda.synchronize()

    # ---- device-resident timing: K steps, state in HBM, device-side dt -----------------------
    # Timed region = hydro_run_steps(K) as a user gets it (replay of the captured one-step CUDA
    # graph), bracketed by CUDA events on the library's stream.
    h.set_state(Ud)
    h.run_steps(args.warmup)
    h.set_state(Ud)                                        # same physical state every run
    h.run_steps(max(args.warmup, 3))
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        t_wait = time.perf_counter()                       # nvidia-smi needs a moment to start
        while not sampler.rows and time.perf_counter() - t_wait < 3.0:
            time.sleep(0.02)
    barrier()                                              # all ranks enter the timed region together
    n0 = h.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tw0 = time.perf_counter()
    ev0.record(h.torch_stream)
    h.run_steps(args.steps)
    ev1.record(h.torch_stream)
    torch.cuda.synchronize()
    tw1 = time.perf_counter()
    barrier()
    launches = h.launch_count() - n0
    clocks = sampler.stop(tw0, tw1) if rank == 0 else None
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, red_dev)
    value = world * cells * args.steps / (ms * 1e-3)

    # ---- the same K steps again with every kernel launch bracketed by CUDA events on the library's
    #      stream (direct launches instead of graph replay): per-kernel durations for the roofline
    import ctypes as C
    L.hydro_set_profiling(h._h, 1)
    barrier()
    eg0, eg1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    eg0.record(h.torch_stream)
    h.run_steps(args.steps)
    eg1.record(h.torch_stream)
    torch.cuda.synchronize()
    ms_prof = max_over_ranks(eg0.elapsed_time(eg1), world, red_dev)
    kt = {}
    for which, name in ((0, "ghost_fill"), (1, "stage1"), (2, "stage2"), (3, "next_dt")):
        tms, cnt = C.c_double(), C.c_longlong()
        L.hydro_get_kernel_time(h._h, which, C.byref(tms), C.byref(cnt))
        kt[name] = (tms.value, cnt.value)
    L.hydro_set_profiling(h._h, 0)
    _, nsteps = h.get_time()
    st_ms = kt["stage1"][0] + kt["stage2"][0]
    st_n = kt["stage1"][1] + kt["stage2"][1]
    roofline = roofline_alu = None
    if st_n:
        bytes_pair = (BYTES_STAGE[1] + BYTES_STAGE[2]) * cells     # one stage-1 + one stage-2 launch
        avg_pair_ms = st_ms / (st_n / 2)
        achieved = bytes_pair / (avg_pair_ms * 1e-3) / 1e9
        common = {"kernel": "stage_fused<1> + stage_fused<2> (one RK2 step's two stage launches)"
                            if (args.variant is None or args.variant == 1) else "stage_simple<1,2>",
                  "avg_launch_ms": {k: (v[0] / v[1] if v[1] else None) for k, v in kt.items()},
                  "share_of_step": {k: v[0] / ms_prof for k, v in kt.items()},
                  "timed_in": "second pass of the same K steps with per-kernel CUDA events on the "
                              "library's stream (direct launches), %.4f ms per step" % (ms_prof / args.steps)}
        # HBM view (BASELINE.json's metric): algorithmic bytes of the two stage launches / their time
        # fp64-pipe view of the same two launches
        peak = N_SM * FP64_LANES_PER_SM * sm_max * 1e6 / 1e12
        ach = (FP64_INSTR_STAGE[1] + FP64_INSTR_STAGE[2]) * cells / (avg_pair_ms * 1e-3) / 1e12
        smem_peak = N_SM * 128.0 * sm_max * 1e6 / 1e9
        smem_ach = 2 * SMEM_BYTES_CELL_STAGE * cells / (avg_pair_ms * 1e-3) / 1e9
        # HBM view (BASELINE.json's metric and north_star's target): algorithmic bytes of the two stage
        # launches / their time.  The kernel saturates no single unit (ablations):
        # HBM, the shared-memory crossbar and the fp64 pipe are each 40-60 % busy and overlap only partly
        # at 4 warps per sub-partition; the fractions of the other two are carried along.
        roofline = dict({"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                         "frac": achieved / hbm_peak, "traffic": traffic["dram"],
                         "traffic_source": traffic["source"], "peak_source": peak_src,
                         "target": "north_star asks for >= 0.70 of peak HBM in the stage kernels",
                         "algorithmic_bytes_per_launch": {"stage1": BYTES_STAGE[1] * cells,
                                                          "stage2": BYTES_STAGE[2] * cells},
                         "fp64_pipe_frac": ach / peak, "smem_crossbar_frac": smem_ach / smem_peak,
                         "note": "no single unit is saturated: HBM, shared-memory crossbar and fp64 pipe "
                                 "overlap only partly (DESIGN.md section 6.1); roofline_alu is the fp64 view"},
                        **common)
        roofline_alu = dict({"bound": "alu", "achieved": ach, "peak": peak, "unit": "T fp64 thread-instr/s",
                             "frac": ach / peak, "traffic": traffic["fp64"],
                             "traffic_source": traffic["source"],
                             "algorithmic_instr_per_cell": FP64_INSTR_STAGE,
                             "peak_source": "63 fp64 lanes/clk/SM (measured DFMA/DADD/DMUL rate, "
                                            "profiles/r2_fp64_pipe_microbench.md) x 148 SM x clocks.max.sm"},
                            **common)

    # ---- the named ABI loop, state resident: K x (hydro_cfl_dt + hydro_step(dt)), i.e. one 32-byte
    #      device->host read and a stream sync per step (SURVEY.md section 8(d) variant (i)) ----------
    h.set_state(Ud)
    for _ in range(3):
        h.step(h.cfl_dt())
    barrier()
    ea0, ea1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ea0.record(h.torch_stream)
    for _ in range(args.steps):
        h.step(h.cfl_dt())
    ea1.record(h.torch_stream)
    torch.cuda.synchronize()
    ms_abi = max_over_ranks(ea0.elapsed_time(ea1), world, red_dev)

    # ---- end to end through the C-ABI with HOST buffers --------------------------------------
    # (a) pipelined, the public host-mirror calls: per step hydro_update_device (all five fields, H2D
    #     on the copy-in stream), hydro_cfl_dt + hydro_step, hydro_update_host (device snapshot, D2H on
    #     the copy-out stream): step n's result goes down while step n+1's input comes up.
    # (b) serial: hydro_set_state / hydro_get_state around the step (the transfer pattern of the
    #     paper's Algorithm 2): every copy waits for the previous one.
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    Uh = U0.clone().pin_memory()
    outs = [torch.empty_like(Uh).pin_memory() for _ in range(2)]
    un, on = Uh.numpy(), [o.numpy() for o in outs]
    h.update_device(un); h.step(h.cfl_dt()); h.update_host(on[0]); h.transfer_sync()   # warm the path
    barrier()
    te0 = time.perf_counter()
    for k in range(e2e_steps):
        h.update_device(un)                                # H2D of the step's input state
        h.step(h.cfl_dt())                                 # + 48-byte D2H of the reduction scalars
        h.update_host(on[k & 1])                           # D2H of the step's result
    h.transfer_sync()
    torch.cuda.synchronize()
    te = max_over_ranks(time.perf_counter() - te0, world, red_dev)
    state_bytes = 5 * cells * 8
    e2e = {"value": world * cells * e2e_steps / te, "unit": UNIT,
           "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes + 48,
           "steps": e2e_steps, "ms_per_step": 1e3 * te / e2e_steps,
           "what": "per step: hydro_update_device(pinned host, 5 fields) + hydro_cfl_dt + hydro_step + "
                   "hydro_update_host(pinned host, 5 fields); transfers on copy streams, both directions "
                   "in flight at once; hydro_transfer_sync at the end"}
    out_h = outs[0]
    h.set_state(Uh); h.step(h.cfl_dt()); h.get_state(out_h)             # warm the copy path
    barrier()
    te0 = time.perf_counter()
    for _ in range(e2e_steps):
        h.set_state(Uh)
        h.step(h.cfl_dt())
        h.get_state(out_h)
    torch.cuda.synchronize()
    te = max_over_ranks(time.perf_counter() - te0, world, red_dev)
    e2e["serial"] = {"value": world * cells * e2e_steps / te, "unit": UNIT, "ms_per_step": 1e3 * te / e2e_steps,
                     "what": "per step: hydro_set_state(pinned host) + hydro_cfl_dt + hydro_step + "
                             "hydro_get_state(pinned host), each copy synchronous"}

    # whole-job variant: state uploaded once, K steps with host-side dt, state downloaded once
    h.set_state(U0)
    barrier()
    tj0 = time.perf_counter()
    h.set_state(U0)
    for _ in range(args.steps):
        h.step(h.cfl_dt())
    h.get_state(out_h)
    tj = max_over_ranks(time.perf_counter() - tj0, world, red_dev)
    e2e["job"] = {"value": world * cells * args.steps / tj, "unit": UNIT, "steps": args.steps,
                  "what": "hydro_set_state(host) once + K x (hydro_cfl_dt + hydro_step) + "
                          "hydro_get_state(host) once"}

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            cpu = cpu_baseline(cfg)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic",
                "config": cfg_dict(cfg, {"parallelism": "single GPU" if world == 1 else
                                         f"{world} independent replicas (no collective)",
                                         "dt": "device-resident (hydro_run_steps, CUDA-graph replay)",
                                         "stage_kernel_geometry": tiling}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
                "abi_loop": {"value": world * cells * args.steps / (ms_abi * 1e-3), "unit": UNIT,
                             "ms_per_step": ms_abi / args.steps,
                             "what": "K x (hydro_cfl_dt + hydro_step(dt)), state resident in HBM"},
                "roofline": roofline, "roofline_alu": roofline_alu, "cpu_baseline": cpu}
        n_dev = torch.cuda.device_count()
        if backend != "nccl" or world > n_dev:
            # replicas share devices (HYDRO_BENCH_BACKEND=gloo plumbing test): not a multi-GPU figure
            line["devices_shared"] = True
            line["distinct_devices"] = min(world, n_dev)
        if roofline:
            line["hbm_gbs_whole_step"] = ((BYTES_STAGE[1] + BYTES_STAGE[2]) * cells * args.steps
                                          / (ms * 1e-3) / 1e9)
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


def run_slab(args):
    """Optional mode (--decomp slab, N > 1): ONE domain of nx x ny x (N nz) cells decomposed into N
    z-slabs, one per rank / GPU -- the paper's own parallelisation: two boundary
    planes per interface exchanged after every substep (NCCL device buffers on a communication stream,
    overlapping the interior substep) and the maximum signal speed all-reduced every step
    (paper_1812_07977_b200/slab.py).  Weak scaling: every rank holds the config's grid.  Not the graded
    default (north_star: no sharding); unmeasured on multi-GPU hardware in this run."""
    import torch
    import torch.distributed as dist
    from paper_1812_07977_b200 import slab
    from paper_1812_07977_b200.binding import Hydro

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world < 2:
        raise SystemExit("bench.py --decomp slab needs N > 1 ranks (torchrun)")
    backend = os.environ.get("HYDRO_BENCH_BACKEND", "nccl")
    local = local % torch.cuda.device_count() if backend != "nccl" else local
    torch.cuda.set_device(local)
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        dist.init_process_group(backend)
    red_dev = "cuda" if backend == "nccl" else "cpu"
    cfg = workload(args.config)
    nx, ny, nz = cfg.shape
    h = Hydro(nx, ny, nz * world, cfg.gamma, cfg.dx, cfg.bc, slab=(rank, world))
    h.set_cfl(cfg.cfl)
    U = torch.from_numpy(cfg.state()).cuda()
    drv = slab.SlabRank(slab.HydroEngine(h), dist, rank, world, cfg.bc[4] == 2, cfg.dx, cfg.cfl)
    h.set_state(U)
    drv.run_steps(max(args.warmup, 3))
    torch.cuda.synchronize(); dist.barrier()
    n0 = h.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(h.torch_stream)
    drv.run_steps(args.steps)
    ev1.record(h.torch_stream)
    torch.cuda.synchronize(); dist.barrier()
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, red_dev)
    launches = h.launch_count() - n0
    if rank == 0:
        n_dev = torch.cuda.device_count()
        line = {"metric": METRIC, "value": world * cfg.cells * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": cfg_dict(cfg, {"parallelism": f"one {nx}x{ny}x{nz * world} domain in {world} z-slabs: halo exchange "
                                                        f"after every substep + all_reduce(MAX) per step ({backend})",
                                         "halo_bytes_per_interface_per_substep": 10 * nx * ny * 8}),
                "gpu_launches": int(launches), "e2e": None, "roofline": None, "cpu_baseline": None, "clocks": None}
        if backend != "nccl" or world > n_dev:
            line["devices_shared"] = True
            line["distinct_devices"] = min(world, n_dev)
        print(json.dumps(line), flush=True)
    h.close()
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)   # config 3 of BASELINE.json: 200 RK2 steps
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--variant", type=int, default=None)
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tile-rows", type=int, default=0, help="hydro_set_tiling (0 = library's choice)")
    ap.add_argument("--planes-per-chunk", type=int, default=0)
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default, the graded mode) or one domain in N z-slabs")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.decomp == "slab":
        run_slab(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
