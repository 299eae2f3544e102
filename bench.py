"""bench.py -- cell-updates/s (fp64) of the shallow-water step loop on B200, with its HBM roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--scale 1.0]

One bench "step" = `--time-steps` (default 100) consecutive time steps of the whole hot path (S0..S4 of
include/swe.h: dt, edge fluxes, limiter, gather, update + friction, CFL reduction) over the whole mesh, enqueued by
ONE swe_step call (CUDA-graph launches, no host synchronisation inside).  Workload: BASELINE.json configs[3], the
~4M-cell river-reach flood wave with wetting/drying (the workload the north_star's target is quoted on), seeded
synthetic (workloads/configs.py).  metric = cell-updates/s = cells x time steps / device time.

N > 1 (torchrun): the path is single-GPU by design ("replicas only"): every rank steps its
own replica of the same workload, no data-path collective; value = all ranks' cell-updates / max-over-ranks time.

--impl reference: the oracle (oracle/, plain single-threaded C++) timed on the host cores on the same workload;
one step = ONE time step of the whole mesh (a bounded sample of the 100-time-step step above).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel come from profiles/ncu_traffic.csv: one row per
# committed `ncu --set full` capture, keyed by kernel name, cell count AND the git blob hash of the source file the
# kernel was compiled from at capture time -- a row whose hash is not the hash of that file as it stands is ignored
# ("traffic": null), so the figure can never describe another kernel than the one being timed
KERNEL_SOURCE = {"k_patch_step": "paper_2102_12862_b200/csrc/swe_patch2_kernel.cuh",
                 "k_edge_flux": "paper_2102_12862_b200/csrc/swe_kernels.cuh",
                 "k_theta_lazy": "paper_2102_12862_b200/csrc/swe_kernels.cuh",
                 "k_cell_update": "paper_2102_12862_b200/csrc/swe_kernels.cuh",
                 "k_step_control": "paper_2102_12862_b200/csrc/swe_kernels.cuh"}


def git_blob_hash(path):
    """sha1 of `blob <size>\0<content>`: what `git hash-object` prints, computed without git."""
    import hashlib
    data = open(os.path.join(ROOT, path), "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_traffic(kernel, n_cells):
    """(bytes per launch, capture name) of the newest matching row of profiles/ncu_traffic.csv, else (None, None)."""
    import csv
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    src = KERNEL_SOURCE.get(kernel)
    if not os.path.exists(path) or src is None:
        return None, None
    want = git_blob_hash(src)
    hit = (None, None)
    for row in csv.DictReader(line for line in open(path) if not line.startswith("#")):
        if row["kernel"] == kernel and int(row["n_cells"]) == int(n_cells) and row["source_blob"] == want:
            hit = (float(row["dram_bytes_per_launch"]), row["capture"])
    return hit


# --morph: parameter sets of swe_set_morphology (formula, alpha, theta_cr, s, d_m, porosity)
MORPH_PARAMS = {1: (1, 0.001, 0.0, 2.65, 1e-3, 0.4), 2: (2, 8.0, 0.047, 2.65, 0.005, 0.4)}
METRIC = "cell_updates_per_s"
UNIT = "cell-updates/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs[id-1]")
    ap.add_argument("--scale", type=float, default=1.0, help="cell-count scale of the workload (1.0 = as named)")
    ap.add_argument("--time-steps", type=int, default=100, help="time steps per bench step (our arm)")
    ap.add_argument("--variant", type=int, default=0, help="include/swe.h SWE_VARIANT_* (0 = library default)")
    ap.add_argument("--patch-cells", type=int, default=0, help="cells per patch of the fused step (0 = default)")
    ap.add_argument("--renumber", type=int, default=1, help="SWE_RENUMBER_*: 0 input order, 1 Morton, 2 RCM")
    ap.add_argument("--shuffle-input", action="store_true", help="randomly renumber the input mesh first (A/B runs)")
    ap.add_argument("--stage", type=float, default=None,
                    help="config 4 only: initial water level relative to the sloped datum (default -2 = the configuration)")
    ap.add_argument("--species", type=int, default=0, help="passive scalar species advected with the flow (0..5)")
    ap.add_argument("--morph", type=int, default=0, choices=[0, 1, 2],
                    help="mobile bed (swe_set_morphology): 1 Grass-like alpha = 0.001, 2 MPM-like alpha = 8, d_m = 5 mm")
    ap.add_argument("--precision", default="double", choices=["double", "single"],
                    help="arithmetic of the step (include/swe.h SWE_PRECISION_*; single: fp32 records and arithmetic in both step variants, DESIGN.md R-21)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-omp", action="store_true", help="also time the oracle source built with OpenMP on all host cores")
    ap.add_argument("--parity-steps", type=int, default=5,
                    help="time steps of the oracle window started from the state after the timed region (0 = off)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-all-wet", action="store_true", help="skip the second (all-wet mesh) line")
    ap.add_argument("--no-other-variant", action="store_true", help="skip the other step variant's line")
    ap.add_argument("--profile-steps", type=int, default=64, help="event-bracketed steps for the roofline object")
    return ap.parse_args()


def peaks():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_workload(config_id, scale, rank=0, world=1, barrier=None, stage=None):
    """Seeded synthetic workload; rank 0 generates, the others read its cache file (generation is ~50 s at 4M)."""
    from workloads import configs as C
    if stage is not None and config_id == 4:
        return C.config4(target_cells=int(4_000_000 * scale), length=10000.0 * scale, stage=stage)
    if world == 1:
        return C.by_id(config_id, scale)
    import pickle
    path = f"/tmp/swe_b200_workload_c{config_id}_s{scale:g}_{os.environ.get('MASTER_PORT', '0')}.pkl"
    if rank == 0:
        w = C.by_id(config_id, scale)
        meta, w.meta = w.meta, {}
        with open(path + ".tmp", "wb") as f:
            pickle.dump(w, f, protocol=4)
        os.replace(path + ".tmp", path)
        w.meta = meta
        barrier()
    else:
        barrier()
        with open(path, "rb") as f:
            w = pickle.load(f)
    barrier()
    if rank == 0:
        try:
            os.remove(path)
        except OSError:
            pass
    return w


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    def __init__(self, index, period=0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
            getattr(nv, "nvmlClocksEventReasonApplicationsClocksSetting", 0x2): "applications_clocks_setting",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def max_over_ranks(x, world, device):
    """Max of a host float over all ranks (the N > 1 timing rule); identity when world == 1."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def aggregate_value(n_cells, time_steps, steps, world, seconds):
    """Whole-job cell-updates/s: every rank advances its own replica (weak scaling, no data-path collective)."""
    return world * n_cells * time_steps * steps / seconds


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def pin_to_one_core():
    """Pins this process to one of the cores it may run on (the oracle is timed single-threaded on a
    pinned core); returns (core, previous affinity) or (None, None) where the platform has no such call."""
    try:
        prev = os.sched_getaffinity(0)
        core = sorted(prev)[-1]
        os.sched_setaffinity(0, {core})
        return core, prev
    except (AttributeError, OSError):
        return None, None


def unpin(prev):
    if prev:
        try:
            os.sched_setaffinity(0, prev)
        except OSError:
            pass


def oracle_time(w, n_warm, max_steps, min_seconds, cfl, morph=0, omp=False, precision="double"):
    """The oracle as it stands on this box's host cores: (cell-updates/s, time steps timed, s).  omp=False: single
    thread (the caller pins the process to one core); omp=True: the same source built with OpenMP, all cores."""
    from oracle import swe_ref
    o = swe_ref.RefSolver(w, omp=omp, precision=precision)
    if morph:
        o.set_morphology(*MORPH_PARAMS[morph])
    if n_warm:
        o.step(n_warm, float("inf"), cfl)
    done, t0 = 0, time.perf_counter()
    while done < max_steps:
        o.step(1, float("inf"), cfl)
        done += 1
        if time.perf_counter() - t0 >= min_seconds:
            break
    dt = time.perf_counter() - t0
    o.close()
    return w.n_cells * done / dt, done, dt


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores; one step = one time step of the whole mesh."""
    if rank != 0:
        return
    from oracle import swe_ref
    w = load_workload(args.config, args.scale)
    core, prev_aff = pin_to_one_core()
    o = swe_ref.RefSolver(w, precision=args.precision)
    if args.morph:
        o.set_morphology(*MORPH_PARAMS[args.morph])
    for _ in range(args.warmup):
        o.step(1, float("inf"), w.cfl)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(1, float("inf"), w.cfl)
    dt = time.perf_counter() - t0
    o.close()
    unpin(prev_aff)
    value = w.n_cells * args.steps / dt
    sample = (f"all {w.n_cells} cells x 1 time step per step (the GPU arm's step is {args.time_steps} time steps); "
              f"single thread pinned to core {core}")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.precision == "double" else "f32", "data": "synthetic",
        "config": {"workload": w.name, "baseline_config": args.config, "n_cells": w.n_cells, "n_edges": w.n_edges,
                   "time_steps_per_step": 1, "cfl": w.cfl, "morph": args.morph, "precision": args.precision},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def parity_window(s, w, info, n_steps, precision="double"):
    """State after the timed region -> oracle (get_state -> set_state at the same t), then n_steps on both sides;
    every cell compared at the north_star tolerances (|d| <= 1e-10 |ref| + 1e-14 max|ref|; dt <= 1e-12 relative;
    identical wet/dry masks).  The oracle runs here as the checker of the timed state, outside every timed region."""
    from oracle import swe_ref
    st = s.get_state()
    o = swe_ref.RefSolver(w, precision=precision)
    o.set_state(*st, t0=info["t"])
    s.set_state(*st, t0=info["t"])
    ig, io = s.step(n_steps, float("inf"), w.cfl), o.step(n_steps, float("inf"), w.cfl)
    got, want = s.get_state(), o.get_state()
    o.close()
    ok = bool(np.array_equal(got[0] > w.h_dry, want[0] > w.h_dry))
    max_rel = 0.0
    for a, b in zip(got, want):
        scale = float(np.max(np.abs(b))) if b.size else 0.0
        err = np.abs(a - b)
        ok = ok and bool(np.all(err <= 1e-10 * np.abs(b) + 1e-14 * scale))
        big = np.abs(b) > 1e-8 * scale
        if np.any(big):
            max_rel = max(max_rel, float(np.max(err[big] / np.abs(b[big]))))
    dt_rel = abs(ig["dt_last"] - io["dt_last"]) / io["dt_last"] if io["dt_last"] else 0.0
    ok = ok and dt_rel <= 1e-12 and ig["n_wet"] == io["n_wet"]
    return {"parity_steps": n_steps, "parity_from_step": info["steps_done"], "parity_ok": ok, "max_rel_err": max_rel,
            "dt_rel_err": dt_rel, "bit_identical": bool(all(np.array_equal(a, b) for a, b in zip(got, want)))}


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    import paper_2102_12862_b200 as P
    P.lib()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    w = load_workload(args.config, args.scale, rank, world, barrier, stage=args.stage)
    if args.shuffle_input:
        w = w.permuted(12862)[0]
    N, E, T = w.n_cells, w.n_edges, args.time_steps
    t_create = time.perf_counter()
    s = P.from_workload(w, device=f"cuda:{local_rank}", variant=args.variant, patch_cells=args.patch_cells,
                        renumber=args.renumber, n_species=args.species, morphology=bool(args.morph),
                        precision=P.PRECISION_SINGLE if args.precision == "single" else P.PRECISION_DOUBLE)
    if args.species:
        from workloads import mesh as WM
        ctr = WM.centroids(w.node_xy, w.tri)
        span = np.ptp(ctr, axis=0) + 1e-300
        phi = [0.5 + 0.5 * np.sin((k + 1) * 6.283185307179586 * (ctr[:, 0] / span[0] + ctr[:, 1] / span[1]))
               for k in range(args.species)]
        s.set_scalars(np.stack([p_ * w.h for p_ in phi]))
        for sid, typ, _ in w.strings:
            if typ == 1:
                s.set_boundary_scalar(sid, [1.0] * args.species)
    if args.morph:
        s.set_morphology(*MORPH_PARAMS[args.morph])
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t_create
    stream = torch.cuda.current_stream(dev)
    s_kernels, patch_stats, s_workspace_bytes = s.step_kernels(), s.patch_stats(), s.workspace_nbytes

    # ---- device-resident arm: W warm-up steps, then exactly K steps between barrier + synchronize on both sides
    for _ in range(args.warmup):
        s.step(T, float("inf"), w.cfl, info=False)
    torch.cuda.synchronize()
    barrier()
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    launches0 = s.kernel_launches
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]    # one chunk = one bench step
    torch.cuda.synchronize()
    ev0.record(stream)
    marks[0].record(stream)
    for k in range(args.steps):
        s.step(T, float("inf"), w.cfl, info=False)
        marks[k + 1].record(stream)
    ev1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    barrier()
    ms = ev0.elapsed_time(ev1)
    chunk_ms = [marks[k].elapsed_time(marks[k + 1]) for k in range(args.steps)]
    ms_median = float(np.median(chunk_ms)) if chunk_ms else None
    launches = s.kernel_launches - launches0
    info = s.step(0, float("inf"), w.cfl, info=True)       # state check after the timed region: finite, mass balance
    # ... and parity: the oracle continues from the GPU's state for a short window (rank 0, N = 1), all cells compared
    parity = None
    if rank == 0 and world == 1 and args.parity_steps > 0 and not args.species and not args.morph:
        parity = parity_window(s, w, info, args.parity_steps, args.precision)
        info = s.step(0, float("inf"), w.cfl, info=True)
    ms = max_over_ranks(ms, world, dev)
    value = aggregate_value(N, T, args.steps, world, ms * 1e-3)

    # ---- roofline of the dominant kernel: event-bracketed kernels inside the library (rank 0)
    roofline = None
    kernel_ms = None
    if rank == 0:
        skipped0 = s.patch_stats()["patch_steps_skipped"]
        kernel_ms = s.profile_step(args.profile_steps, w.cfl)
        st = s.patch_stats()
        # fused patch step: blocks that find their whole patch dry move no mesh data; their share of the launch is
        # taken OUT of the algorithmic bytes (never counted as achieved bandwidth)
        f_skip = (st["patch_steps_skipped"] - skipped0) / max(1, args.profile_steps * max(1, st["patches"]))
        alg = {k: v * (1.0 - f_skip) if k == "k_patch_step" else v for k, v in s.algorithmic_bytes().items()}
        # SURVEY.md section 8(d) "Algorithmic bytes per cell-step" (132 B one-pass, 284 B = 148 + 136 two-kernel) x the cells
        # the launch actually processes: the basis of `achieved` / `frac`; the library's own count (32-byte records,
        # DESIGN.md section 6) gives `frac_own_count`
        surv = {k: v * (1.0 - f_skip) if k == "k_patch_step" else v for k, v in s.survey_bytes().items()}
        top = max(kernel_ms, key=kernel_ms.get)
        peak, how = peaks()
        achieved = surv[top] / (kernel_ms[top] * 1e-3) / 1e9
        achieved_own = alg[top] / (kernel_ms[top] * 1e-3) / 1e9
        traffic, capture = ncu_traffic(top, N)
        roofline = {"bound": "hbm", "kernel": top, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": traffic, "traffic_capture": capture, "peak_source": how,
                    "bytes_basis": "SURVEY.md 8(d): %d B per cell-step x cells processed" % round(surv[top] / max(1.0, N * (1.0 - (f_skip if top == "k_patch_step" else 0.0)))),
                    "algorithmic_bytes_per_launch": surv[top], "kernel_ms": kernel_ms[top],
                    "frac_own_count": achieved_own / peak, "achieved_own_count": achieved_own,
                    "own_count_bytes_per_launch": alg[top],
                    "dry_patch_fraction_skipped": f_skip,
                    "step_algorithmic_bytes": sum(surv.values()),
                    "step_achieved": sum(surv.values()) / (ms * 1e-3 / (T * args.steps)) / 1e9,
                    "share_of_step": kernel_ms[top] / sum(kernel_ms.values())}
        if top == "k_patch_step":
            roofline["note"] = ("the fused patch step moves about a third of the bytes of the bandwidth-bound "
                                "three-pass step (other_variant: its kernels and whole step against the same HBM "
                                "peak) and is bound by fp64 issue / latency, not by HBM (DESIGN.md section 7)")
        if args.morph and top == "k_edge_flux":
            roofline["traffic"] = None
            roofline["note"] = ("mobile bed: the <kMorph> edge kernel is bound by fp64 instruction issue (Table 2 + Eq. 16 "
                                "per side on top of the HLLC flux; ncu: fp64 pipe 47 %, issue slots 58 % at 24 warps/SM), "
                                "not by HBM (profiles/r1j_morph.md)")

    # ---- end-to-end arm: the same K steps through the C-ABI with HOST (pinned) buffers, copies inside the region
    e2e = None
    if not args.no_e2e:
        host = [torch.empty(N, dtype=torch.float64, pin_memory=True).numpy() for _ in range(3)]
        s.get_state(tuple(host))
        host_q = s.get_scalars() if args.species else None      # (pageable; the scalar copies are in the region too)
        t_now = info["t"]
        for _ in range(min(2, args.warmup)):
            s.set_state(*host, t0=t_now)
            t_now = s.step(T, float("inf"), w.cfl, info=True)["t"]
            s.get_state(tuple(host))
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            s.set_state(*host, t0=t_now)                               # H2D: 3 x 8 x N bytes
            if args.species:
                s.set_scalars(host_q)                                  # H2D: species x 8 x N bytes
            t_now = s.step(T, float("inf"), w.cfl, info=True)["t"]    # info: the step's result scalars come back
            s.get_state(tuple(host))                                   # D2H: 3 x 8 x N bytes
            if args.species:
                host_q = s.get_scalars()
        torch.cuda.synchronize()
        dt_e2e = time.perf_counter() - t0
        dt_e2e = max_over_ranks(dt_e2e, world, dev)
        e2e = {"value": aggregate_value(N, T, args.steps, world, dt_e2e), "unit": UNIT, "h2d_bytes_per_step": (24 + 8 * args.species) * N,
               "d2h_bytes_per_step": (24 + 8 * args.species) * N + 72}
    s.close()

    # ---- the other step variant on the same workload (rank 0, N = 1): the default is the fused patch step, which
    # moves a third of the bytes; the three-pass step (edge flux -> theta -> CSR gather/update, the design the
    # north_star names) is the bandwidth-bound one, so its per-kernel HBM fractions are reported beside the default's
    other = None
    if rank == 0 and world == 1 and not args.no_other_variant and args.variant == 0 and args.species == 0 and not args.morph:
        ov = P.VARIANT_THREE_PASS if s_kernels[-1] == "k_patch_step" else P.VARIANT_PATCH
        s3 = P.from_workload(w, device=f"cuda:{local_rank}", variant=ov, renumber=args.renumber,
                             precision=P.PRECISION_SINGLE if args.precision == "single" else P.PRECISION_DOUBLE)
        for _ in range(2):
            s3.step(T, float("inf"), w.cfl, info=False)
        torch.cuda.synchronize()
        ev0.record(stream)
        for _ in range(5):
            s3.step(T, float("inf"), w.cfl, info=False)
        ev1.record(stream)
        torch.cuda.synchronize()
        ms3 = ev0.elapsed_time(ev1)
        km3 = s3.profile_step(16, w.cfl)
        alg3 = s3.survey_bytes()
        pk = peaks()[0]
        other = {"step_kernels": s3.step_kernels(), "value": N * T * 5 / (ms3 * 1e-3), "unit": UNIT,
                 "ms_per_time_step": ms3 / (5 * T), "kernel_ms": km3,
                 "kernel_hbm_frac": {k: (alg3[k] / (km3[k] * 1e-3) / 1e9 / pk if km3[k] > 0 else 0.0) for k in km3},
                 "step_algorithmic_bytes": sum(alg3.values()),
                 "step_achieved_gbs": sum(alg3.values()) / (ms3 * 1e-3 / (5 * T)) / 1e9,
                 "step_hbm_frac": sum(alg3.values()) / (ms3 * 1e-3 / (5 * T)) / 1e9 / pk}
        s3.close()

    # ---- second line (rank 0, N = 1): an ALL-WET mesh of the same size, where no patch can be skipped -- the
    # BASELINE.json configs[4] construction (circular dam break, every cell wet, friction everywhere) at 4M cells
    all_wet = None
    if rank == 0 and world == 1 and not args.no_all_wet and args.species == 0 and not args.morph:
        from workloads import configs as C
        w2 = C.config5(target_cells=N)
        s2 = P.from_workload(w2, device=f"cuda:{local_rank}", variant=args.variant, patch_cells=args.patch_cells,
                             precision=P.PRECISION_SINGLE if args.precision == "single" else P.PRECISION_DOUBLE)
        for _ in range(2):
            s2.step(T, float("inf"), w2.cfl, info=False)
        torch.cuda.synchronize()
        ev0.record(stream)
        for _ in range(5):
            s2.step(T, float("inf"), w2.cfl, info=False)
        ev1.record(stream)
        torch.cuda.synchronize()
        ms2 = ev0.elapsed_time(ev1)
        km2 = s2.profile_step(16, w2.cfl)
        i2 = s2.step(0, float("inf"), w2.cfl, info=True)
        alg2 = s2.survey_bytes()
        top2 = max(km2, key=km2.get)
        all_wet = {"workload": w2.name, "n_cells": w2.n_cells, "value": w2.n_cells * T * 5 / (ms2 * 1e-3), "unit": UNIT,
                   "ms_per_time_step": ms2 / (5 * T), "kernel_ms": km2, "n_wet": i2["n_wet"],
                   "patch_steps_skipped": s2.patch_stats()["patch_steps_skipped"],
                   "roofline_frac": alg2[top2] / (km2[top2] * 1e-3) / 1e9 / peaks()[0], "flags": i2["flags"]}
        s2.close()
        del w2

    # ---- CPU baseline: the oracle, single thread, bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        core, prev_aff = pin_to_one_core()
        v, n_done, secs = oracle_time(w, 1, 40, 12.0, w.cfl, args.morph, precision=args.precision)
        unpin(prev_aff)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"all {N} cells x {n_done} time steps from the initial state ({secs:.1f} s, 1 thread pinned to core {core})"}
        if args.cpu_omp:        # PAPER.md:427 (the `omp` backend): the same oracle source, OpenMP on every host core
            v2, n2, secs2 = oracle_time(w, 1, 40, 8.0, w.cfl, args.morph, omp=True)
            cpu["omp"] = {"value": v2, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle, OpenMP build",
                          "sample": f"all {N} cells x {n2} time steps ({secs2:.1f} s)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "ms_per_step_median": ms_median,
            "ms_per_step_chunks": chunk_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if args.precision == "double" else "f32", "data": "synthetic",
            "config": {"workload": w.name, "precision": args.precision, "baseline_config": args.config, "n_cells": N, "n_edges": E,
                       "time_steps_per_step": T, "cfl": w.cfl, "parallelism": f"replicas x{world}",
                       "l2": "working set (%.0f MB) larger than L2, no flush" % (s_workspace_bytes / 1e6),
                       "create_s": round(t_create, 2), "renumber": args.renumber, "shuffled_input": args.shuffle_input, "n_species": args.species, "morph": args.morph, "stage": args.stage, "step_kernels": s_kernels, "patch": patch_stats},
            "ms_per_time_step": ms / (args.steps * T),
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "kernel_ms": kernel_ms, "cpu_baseline": cpu, "all_wet": all_wet, "other_variant": other,
            "state_check": dict({"t": info["t"], "steps_done": info["steps_done"], "n_wet": info["n_wet"],
                                 "vol_clipped": info["vol_clipped"], "flags": info["flags"]}, **(parity or {})),
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
