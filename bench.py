"""bench.py — zone-updates/s of one full AGATE finite-volume MHD time step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

A "step" is one pass of the whole hot path over the resident state: Courant reduction (A7), then per Runge-Kutta
stage ghost fill (A0) + the fused stage kernel (A1-A6).  On 3-D grids A7 of step n+1 runs inside the last stage of
step n and the step starts with a one-thread kernel that turns that v_max into dt.  Default workload: BASELINE.json config 5 (3D ideal MHD,
512^3, PLM + eq.4 beta=1.3, HLLD, SSP-RK2, seeded synthetic state) on one GPU.  N > 1 runs N
independent replicas of that problem, one per rank (the path is single-GPU by specification: "replicas only",
weak scaling, no data-path collective); timing = barrier + device events, max over ranks.

The JSON line carries: value (device-resident throughput), e2e (through the C-ABI with pinned HOST buffers, the
full state copied in and out every step), roofline (dominant kernel = the fused stage kernel, bound = FP64 ALU
pipe), cpu_baseline (the oracle, as it stands, on a bounded sample), clocks, gpu_launches.

--impl reference times the CPU oracle (oracle/) on the box's host cores on a bounded sample of the same workload.
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

METRIC = "zone-updates/sec per full step (fp64)"
UNIT = "zone-updates/s"

# Algorithmic flop per zone per full step (both stages + dt reduction), SURVEY §8(d) convention (add/sub/mul/
# compare/min/max/div/sqrt = 1, FMA = 2): the lean hand count of SURVEY §8(d); the oracle's
# own as-written count (oracle.count_ops) is higher (1774 / 2265 / 3350 / 2072 / 3292) because it evaluates both
# sides' fluxes and divides where a shared reciprocal serves.  The smaller figure is used so the fraction is not
# flattered.
# config 6 (Orszag-Tang + GLM, NEXT-1): config 1's 2-D HLL count + 120 for the ninth variable (slopes, 2x2 face
# problem, flux difference, source)
# config 7 (Orszag-Tang in CGL MHD, NEXT-2): the oracle's as-written count (2098, oracle.count_ops) scaled by config
# 1's lean / as-written ratio (1430 / 1774)
# config 8 (3-D Hall, not a BASELINE.json config): the oracle's as-written count (3202) scaled by config 4's lean /
# as-written ratio (1760 / 2072)
# config 9 (CGL + GLM): config 7's count + config 6's 120 for the GLM scalar
FLOP_PER_ZONE_STEP = {1: 1430.0, 2: 1890.0, 3: 2770.0, 4: 1760.0, 5: 2770.0, 6: 1550.0, 7: 1690.0, 8: 2720.0, 9: 1810.0}
FLOP_DT_PER_ZONE = {1: 45.0, 2: 45.0, 3: 45.0, 4: 60.0, 5: 45.0, 6: 45.0, 7: 90.0, 8: 60.0, 9: 90.0}
BYTES_PER_ZONE_STEP = 320.0            # 5 x 8 variables x 8 B; 360 with the GLM scalar (config 6)
# DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum, mean of the two stage
# launches of one step) from `ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum -k regex:stage -s 2 -c 2` on the
# same bench command with the final kernels (profiles/r2_stage3d.md "final traffic"; the full captures in r2_metrics.csv
# were taken a few commits earlier and agree within 1.5 %)
NCU_TRAFFIC_BYTES = {5: 0.5 * (11525812736 + 8910902016 + 20068614912 + 8812694528),
                     2: 0.5 * (283653632 + 225981952 + 558576640 + 226220800),
                     4: 0.5 * (79418368 + 23350016 + 153315328 + 24589824),
                     8: 0.5 * (1412547840 + 1090191616 + 2523881728 + 1086261504),
                     6: 0.5 * (318541568 + 258995200 + 627718400 + 260007936),
                     7: 0.5 * (318549760 + 258905088 + 627584768 + 260304128),
                     9: 0.5 * (374100480 + 297494528 + 739145984 + 299099648)}
# ... and the kernels they were captured on: sha256 over csrc/*.cu* at capture time.  When the kernels have changed
# since, the figure is stale and the line reports "traffic": null instead (profiles/ names the capture).
NCU_TRAFFIC_CSRC_SHA = "2877b02b7181cef3"


def csrc_sha():
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2503_20899_b200", "csrc", "*.cu*"))):
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # 148 SMs x 64 DFMA lanes x 2 x max SM clock = 37.2

# reduced size of the bounded CPU sample per config (same recipe and seed), and its step count
CPU_SAMPLE = {1: (128, 10), 2: (512, 8), 3: (96, 4), 4: (512, 8), 5: (96, 4), 6: (512, 8), 7: (512, 8), 8: (96, 4), 9: (512, 8)}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5, 6, 7, 8, 9],
                    help="1-5: BASELINE.json configs; 6: Orszag-Tang + GLM, the workload of the paper's Table 2; "
                         "7: Orszag-Tang in CGL MHD; 8: Hall MHD on config 3's 3-D recipe")
    ap.add_argument("--to-time", type=float, default=0.0,
                    help="config 6: also run the problem from t=0 to this time (the paper ran to 0.5) and report the "
                         "device wall time beside the paper's A100 figure")
    ap.add_argument("--n", type=int, default=0, help="override the per-dimension resolution (debugging)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--decomp", action="store_true",
                    help="NEXT-4: slab domain decomposition along the last active dimension instead of replicas: every "
                         "rank holds one full-size slab of a domain N times as long (weak scaling), halo exchange per "
                         "stage, one all-reduce(max) per step; at N = 1 the slab is its own periodic neighbour")
    ap.add_argument("--cgl-form", type=int, default=0, choices=[0, 1],
                    help="config 7: 0 = logarithmic A of eq.18 (the paper's preferred form), 1 = A of eq.16 (eqs.24-25)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    return ap.parse_args()


def workload_name(wl):
    return wl.name


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def cpu_oracle_rate(config, steps=None, warmup=0, all_cores=False):
    """The oracle as it stands (single-threaded build default) on a bounded sample; returns dict for the JSON."""
    import oracle
    from workloads import make_workload
    n, nst = CPU_SAMPLE[config]
    if steps is not None:
        nst = steps
    wl = make_workload(config, n=n)
    ref = oracle.RefSolver.from_workload(wl)
    if warmup:
        ref.advance(warmup)
    t0 = time.perf_counter()
    ref.advance(nst)
    dt = time.perf_counter() - t0
    cores1 = oracle.get_threads()
    allc = None
    if all_cores and (os.cpu_count() or 1) > 1:
        # the same loops under OpenMP on every host core (bitwise identical results, tests/test_oracle_pins.py)
        oracle.set_threads(os.cpu_count())
        try:
            ref.set_state(wl.U)
            ref.advance(1)
            t0 = time.perf_counter()
            ref.advance(nst)
            dta = time.perf_counter() - t0
            allc = {"value": wl.zones * nst / dta, "unit": UNIT, "cores": oracle.get_threads(), "cpu": cpu_model()}
        finally:
            oracle.set_threads(1)
    ref.close()
    out = {"value": wl.zones * nst / dt, "unit": UNIT, "cores": cores1, "kind": "oracle",
           "sample": f"config {config} recipe at {wl.shape[0]}^{wl.ndim}, {nst} full steps, "
                     f"{os.cpu_count()} host cores present"}
    if allc is not None:
        out["all_cores"] = allc
    return out, dt / nst, wl


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    base, per_step, wl = cpu_oracle_rate(args.config, steps=args.steps, warmup=args.warmup)
    line = {"metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": f"BASELINE.json config {args.config} (bounded CPU sample: {base['sample']})"},
            "cpu_baseline": base,
            "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def max_over_ranks(x, world, device):
    """Timing rule for N > 1 (replicas only, no data-path collective): every rank times its own K steps on the
    device, the job's time is the MAX over ranks."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(zones_per_rank, world, steps, ms_max):
    """Whole-job zone-updates/s: every rank advanced its own replica (weak scaling) in the slowest rank's time."""
    return zones_per_rank * world * steps / (ms_max * 1e-3)


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the CUDA path has no CPU fallback")
    import paper_2503_20899_b200 as ag
    from workloads import make_workload

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = args.config
    wl = make_workload(cfg, n=args.n or None)
    zones = wl.zones
    over = {}
    if cfg == 9 and args.cgl_form == 1:
        raise SystemExit("--cgl-form 1 is offered for config 7 only: with the GLM scalar on, eq.16's A runs out of the "
                         "physical range at the vortex's field nulls, in the oracle as on the GPU (DESIGN.md section 11)")
    if cfg == 7 and args.cgl_form == 1:
        # input definition of the other thermodynamic variable (eq.16): A = (rho / |B|)^3 p_perp / p_par
        W = wl.W
        b2 = W[5] ** 2 + W[6] ** 2 + W[7] ** 2
        wl.U[8] = (W[0] ** 3 / (b2 * np.sqrt(b2))) * (W[8] / W[4])
        wl.name += " (A of eq.16)"
        over["cgl_form"] = 1
    wl.W = None                                       # only U is needed; frees one state-sized host array
    K, Wm = args.steps, args.warmup
    if args.decomp:
        return run_decomp(args, ag, wl, world, rank, local, dev, barrier)
    sim = ag.Agate.from_workload(wl, device=dev, set_state=False, **over)
    Uh = torch.from_numpy(wl.U).pin_memory()
    info = sim.launch_info()
    fp64_peak = ag.measure_fp64_peak(10)

    # ---- device-resident throughput: K steps, state already in HBM --------------------------------------
    sim.set_state(Uh)
    sim.advance(Wm)                                   # warm-up (also instantiates the CUDA graph)
    sim.set_state(Uh)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(local) as clk:
        e0.record(sim.stream)
        sim.advance(K, sync=False)
        e1.record(sim.stream)
        barrier()
    ms = e0.elapsed_time(e1)
    sim.poll()
    ms_max = max_over_ranks(ms, world, dev)
    value = aggregate_rate(zones, world, K, ms_max)

    # ---- per-launch duration of the dominant kernel (fused stage), CUDA events on its own stream ---------
    sim.set_state(Uh)
    sim.set_timing(True)
    sim.advance(K)
    st_ms, st_n = sim.stage_time()
    sim.set_timing(False)
    stage_ms = st_ms / max(st_n, 1)
    flop_stage = (FLOP_PER_ZONE_STEP[cfg] - FLOP_DT_PER_ZONE[cfg]) / 2.0 * zones
    achieved = flop_stage / (stage_ms * 1e-3) / 1e12
    peaks, peak_src = measured_peaks()
    bytes_step = BYTES_PER_ZONE_STEP * {6: 9.0 / 8.0, 7: 9.0 / 8.0, 9: 10.0 / 8.0}.get(cfg, 1.0)
    hbm_frac = (bytes_step / 5.0 * 2.5 * zones / (stage_ms * 1e-3) / 1e9) / peaks["hbm_gbs"]
    roofline = {"bound": "alu", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": achieved / fp64_peak, "frac_of_nominal": achieved / FP64_NOMINAL_TFLOPS, "traffic": (NCU_TRAFFIC_BYTES.get(cfg) if (not args.n and csrc_sha() == NCU_TRAFFIC_CSRC_SHA) else None),
                "traffic_source": f"ncu --set full capture of kernels with csrc sha {NCU_TRAFFIC_CSRC_SHA} (profiles/); "
                                  f"this run's csrc sha {csrc_sha()}",
                "algorithmic_bytes": bytes_step / 2.0 * zones,
                "kernel": {3: "stage3d_kernel", 2: "stage2d_kernel"}.get(wl.ndim, "stage_kernel"), "ms_per_launch": stage_ms, "launches_timed": st_n,
                "stage_share_of_step": 2.0 * stage_ms * K / ms_max if st_n else None,
                "peak_source": "FP64 DFMA micro-benchmark of this run (agate_measure_fp64_peak); nominal "
                               f"{FP64_NOMINAL_TFLOPS:.1f} = 148 SM x 64 lanes x 2 x 1.965 GHz",
                "hbm_frac_of_" + peak_src: hbm_frac,
                "flop_per_zone_stage": flop_stage / zones}

    # ---- end to end through the C-ABI with HOST buffers: every step copies the state in and out ---------
    e2e = None
    if not args.no_e2e:
        Ke = min(K, 4)
        out = torch.empty_like(Uh).pin_memory()
        sim.set_state(Uh); sim.step(0.0); sim.get_state(out)            # warm-up
        barrier()
        t0 = time.perf_counter()
        a, b = Uh, out
        for _ in range(Ke):
            sim.set_state(a)
            sim.step(0.0, sync=False)
            sim.get_state(b)
            a, b = b, a
        barrier()
        te = time.perf_counter() - t0
        te_max = max_over_ranks(te, world, dev)
        nbytes = Uh.numel() * 8
        e2e = {"value": aggregate_rate(zones, world, Ke, te_max * 1e3), "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "steps": Ke,
               "note": "agate_set_state(host pinned) + agate_step + agate_get_state(host pinned) per step"}

    # ---- config 6: the paper's own run (Table 2): Orszag-Tang + GLM from t = 0 to t_end -------------
    table2 = None
    if cfg == 6 and args.to_time > 0.0 and world == 1:
        sim.set_state(Uh)
        sim.advance(1)                                # graph instantiation outside the timed region
        sim.set_state(Uh)
        e0.record(sim.stream)
        nst, t = 0, 0.0
        while t < args.to_time:
            t = sim.advance(50)
            nst += 50
        e1.record(sim.stream)
        torch.cuda.synchronize()
        paper = {32: 0.27, 64: 0.450, 128: 0.82, 256: 1.55, 512: 3.04, 1024: 12.0, 2048: 87.1}
        table2 = {"t_end": t, "steps": nst, "wall_s": e0.elapsed_time(e1) * 1e-3, "n": wl.shape[0],
                  "paper_kernel_mode_a100_s": paper.get(wl.shape[0]),
                  "note": "paper: whole-run wall clock of AGATE's Kernel mode on one A100 (Table 2, P:L348-354; "
                          "includes start-up and output); here: device time of the stepping only -- context, not a "
                          "like-for-like benchmark"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": (f"BASELINE.json config {cfg}: {wl.name}" if cfg <= 5 else
                                        f"not a BASELINE.json config: {wl.name}"), "zones_per_gpu": zones,
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": "state (2 x %.2f GB) is larger than L2; no flush needed" % (zones * 64 / 1e9)
                                 if zones * 64 > 2.5e8 else "state fits L2 (small config); numbers are L2-resident",
                           "launch": info},
                "roofline": roofline, "clocks": clk.summary(), "gpu_launches": info["launches_per_step"] * K,
                "e2e": e2e}
        if table2 is not None:
            line["paper_table2_run"] = table2
        if not args.no_cpu and world >= 1:
            line["cpu_baseline"] = cpu_oracle_rate(cfg, all_cores=True)[0]
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_decomp(args, ag, wl, world, rank, local, dev, barrier):
    """NEXT-4 arm: one slab per rank (weak scaling: the domain is N slabs long in its last active dimension, every
    slab carries the config's seeded state, which is periodic, so the stacked state is smooth across the cut faces).
    Per step: one all-reduce(max) of the device-resident v_max; per stage: ghost fill, pack, halo exchange (NCCL
    send/recv between neighbours; two device copies when N = 1), unpack, stage kernel."""
    import torch
    import torch.distributed as dist
    from paper_2503_20899_b200 import slab
    if wl.ndim < 2:
        raise SystemExit("--decomp needs a 2-D or 3-D config")
    K, Wm, zones, cfg = args.steps, args.warmup, wl.zones, args.config
    sim = ag.Agate.from_workload(wl, device=dev, set_state=False)
    Uh = torch.from_numpy(wl.U).pin_memory()
    st = slab.SlabStepper(sim, rank, world, True)
    info = sim.launch_info()
    sim.set_state(Uh); st.reset()
    for _ in range(Wm):
        st.step()
    sim.set_state(Uh); st.reset()
    st.step()                                          # the first step takes v_max through the host; time the steady state
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(local) as clk:
        e0.record(sim.stream)
        for _ in range(K):
            st.step()
        e1.record(sim.stream)
        barrier()
    ms = e0.elapsed_time(e1)
    sim.poll()
    ms_max = max_over_ranks(ms, world, dev)
    value = aggregate_rate(zones, world, K, ms_max)
    halo = sim.halo_bytes()
    if rank == 0:
        rk = int(sim.cfg.rk)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"BASELINE.json config {cfg} recipe as one slab per GPU: {wl.name}",
                           "zones_per_gpu": zones,
                           "parallelism": f"slab decomposition along {'z' if wl.ndim == 3 else 'y'} over {world} rank(s): "
                                          "halo exchange per stage (2 layers x all variables per cut face, "
                                          + ("NCCL send/recv" if world > 1 else "device copies: the slab is its own neighbour")
                                          + "), one all-reduce(max) of v_max per step",
                           "halo_bytes_per_face_per_stage": halo, "launch": info},
                "clocks": clk.summary(), "gpu_launches": (1 + 2 * rk) * K,
                "roofline": None, "e2e": None,
                "note": "NEXT-4 arm; the headline line is the default (replicas) arm.  No scaling curve exists until "
                        "this runs on a multi-GPU node."}
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
