"""bench.py -- zone-updates/s per RK substep of the HORIZON GRMHD update on B200 (BASELINE.json metric).

Contract: `python bench.py --gpus N --steps K --warmup W [--impl reference]` prints ONE JSON line.

Workload: BASELINE.json config 5, the Kerr-Schild throughput sweep, at 256^3 in
fp64 -- the grid north_star quotes its target on.  A bench "step" is one full third-order Runge-Kutta
step = 3 substeps through `hz_step(dt, 1)`; every substep is one pass of the whole hot path (rows
a1-a9 of DESIGN.md section 2).  `value` = interior cells x 3 x K / device time of the K steps.  The
resident state (46 fields x 134 MB in fp64) is ~50x the 126 MB L2, so every pass streams from HBM
("inputs larger than L2").  With --gpus N > 1 every rank runs an independent replica of the same
box (no exchange step exists on this path yet), timed as the max over ranks.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores on a
bounded sub-grid of the same workload; it is a reported baseline, not the target.
"""
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

METRIC = "zone-updates/sec per RK substep"
UNIT = "zone-updates/s"
SUBSTEPS_PER_STEP = 3

# Algorithmic words per zone per substep of each kernel, cleaning on.
# whole path: read P(9) + metric(10) + U^(k)(9) + U^n(9, stages 1-2 only -> 6 on average), write U(9) + P(9)
ALGO_WORDS_PATH = 52.0
# Algorithmic flops per zone per substep (flops k_substep executes per zone by ncu,
# 4120 in fp64 and 3190 in fp32, less the ~10 % that is duplicated tile-boundary face work; the plain
# oracle counts 4564 add+mul, 648 div, 59 sqrt).  FMA = 2.
ALGO_FLOPS = {"f64": 3700.0, "f32": 2900.0, "f32h": 2900.0}
# ALU peak (B200_PROFILING.md unit counts): 148 SMs x lanes x 2 flop x max SM clock
SMS, LANES = 148, {"f64": 64, "f32": 128, "f32h": 128}
# ncu dram__bytes_read.sum + dram__bytes_write.sum of one k_substep launch at 128^3, per zone
# (profiles/r01_substep.md); scaled to the launch's zones below
TRAFFIC_BYTES_PER_ZONE = {"f64": 494.0, "f32": 263.0, "f32h": 263.0}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thr = threading.Thread(target=self._read, daemon=True)
        self.thr.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for (t, line) in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                smax = float(f[1])
                if t0 <= t <= t1 or not sm:
                    sm.append(float(f[0]))
                    power.append(float(f[2]))
            except ValueError:
                continue
            if t0 <= t <= t1:
                for nme, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power) if power else None}


def oracle_rate(nsub_grid, steps, warmup):
    """Zone-updates/s per substep of the CPU oracle, as it stands, on a sub-grid of the Kerr sweep."""
    import workloads as wl
    from oracle import Oracle, OracleParams
    from oracle import binding as ob
    w = wl.kerr_sweep(nsub_grid)
    o = Oracle(w.n, w.h, w.bc, OracleParams.default(**w.params))
    o.set_metric(w.alpha, w.beta3, w.gamma6)
    o.set_primitives(w.prim8)
    for _ in range(warmup):
        o.step(w.dt, 1)
    t = time.perf_counter()
    for _ in range(steps):
        o.step(w.dt, 1)
    el = time.perf_counter() - t
    rate = w.ncell * SUBSTEPS_PER_STEP * steps / el
    return rate, el, ob.num_threads(), w.ncell


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n = args.ref_n
    rate, el, cores, ncell = oracle_rate(n, args.steps, min(args.warmup, 1))
    sample = (f"{n}^3 sub-grid of the Kerr-Schild sweep (same generator and seeds as the {args.n}^3 workload), "
              f"{args.steps} full RK3 steps = {args.steps * 3} substeps, fp64, OpenMP over the outer cell loop")
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"kerr_sweep_{args.n}^3 (BASELINE.json config 5), timed on a bounded sample", "grid": [n, n, n],
                   "substeps_per_step": SUBSTEPS_PER_STEP},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def make_workload(wl, name, n):
    """The five BASELINE.json configs at their stated sizes (kerr: n^3, the bench default 256^3)."""
    if name == "kerr":
        return wl.kerr_sweep(n), f"kerr_sweep_{n}^3 (BASELINE.json config 5: Kerr-Schild a=0.9, seeded torus, cleaning on)"
    if name == "tube":
        return wl.shock_tube(400), "shock_tube_400x1x1 (BASELINE.json config 1)"
    if name == "alfven":
        return wl.alfven_wave(64), "alfven_wave_64^3 (BASELINE.json config 2)"
    if name == "blast":
        return wl.blast(128), "blast_128^3 (BASELINE.json config 3)"
    if name == "tov":
        return wl.tov_star(192), "tov_star_192^3 (BASELINE.json config 4)"
    raise ValueError(name)


def max_over_ranks(ms, world, device):
    """Slowest rank's time: the only cross-rank operation of the replica path."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_gpu(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import workloads as wl
    from paper_1102_5202_b200 import Horizon, lib

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the HORIZON update has no CPU fallback")
    lib()  # fails loudly if libhz.so is missing
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    n, dtype = args.n, args.dtype
    K, W = args.steps, max(args.warmup, 3)
    w, wname = make_workload(wl, args.workload, n)
    if args.recon == "ppm":
        import dataclasses
        w = dataclasses.replace(w, params={**w.params, "recon": 1})
        wname += ", PPM reconstruction"
    stream = torch.cuda.current_stream()
    es = 8 if dtype == "f64" else 4
    shard = args.shard and world > 1
    if shard:
        # strong scaling: the ONE global box cut into `world` slabs along z, ghost planes exchanged over
        # NCCL after every substep (paper_1102_5202_b200/slab.py)
        from paper_1102_5202_b200 import DistSlabHorizon
        from paper_1102_5202_b200.binding import HZ_HALO_PRIM
        dsh = DistSlabHorizon(w, dtype=dtype)
        hz = dsh.slab.hz
        step = lambda: dsh.step(w.dt, 1)
        ncell = dsh.slab.ncell                      # this rank's zones
        total_cells = w.ncell                       # whole job
    else:
        hz = Horizon.from_workload(w, dtype=dtype, stream=stream)
        step = lambda: hz.step(w.dt, 1)
        ncell = w.ncell
        total_cells = world * w.ncell               # replicas: every rank a full box

    # ---- device-resident timing: inputs in HBM, K x hz_step(dt, 1) --------------------------------
    for _ in range(W):
        step()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    barrier()
    launches0 = hz.launch_count()
    hz.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(stream)
    for _ in range(K):
        step()
    e1.record(stream)
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    prof = hz.profile_read()
    hz.profile(False)
    launches = hz.launch_count() - launches0
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ms = max_over_ranks(ms, world, "cuda")
    value = total_cells * SUBSTEPS_PER_STEP * K / (ms * 1e-3)
    d = hz.diagnostics()
    finite = all(np.isfinite(v) for v in d.values())

    # ---- end to end through the C ABI with HOST buffers -------------------------------------------
    # every step: hz_set_primitives(pinned host prim8) -> hz_step(dt, 1) -> hz_get_primitives(pinned host)
    td = torch.float64 if dtype == "f64" else torch.float32
    h_in = torch.from_numpy(hz.get_primitives()).to(td).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    Ke = max(1, min(K, args.e2e_steps))
    def e2e_step():
        hz.set_primitives(h_in)
        if shard:
            dsh.tr.exchange(dsh.slab, HZ_HALO_PRIM)
        step()
        hz.get_primitives(out=h_out)

    for _ in range(2):
        e2e_step()
    barrier()
    e0.record(stream)
    for _ in range(Ke):
        e2e_step()
    e1.record(stream)
    barrier()
    ms_e = e0.elapsed_time(e1)
    ms_e = max_over_ranks(ms_e, world, "cuda")
    e2e_value = total_cells * SUBSTEPS_PER_STEP * Ke / (ms_e * 1e-3)
    assert bool(torch.isfinite(h_out).all()), "non-finite primitives after the end-to-end steps"

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel ------------------------------------
    # The path is bound by plain ALU arithmetic in both precisions (ALU bound 10.1 / 25.7 G zone-updates/s
    # against 15.7 / 31.4 G for HBM), so the roofline is "alu"; the HBM view is reported beside it.
    hbm_gbs, peak_src, sm_max = peaks()
    tot_ms = sum(v[0] for v in prof.values())
    dom = max(prof, key=lambda k: prof[k][0])
    dom_ms, dom_n = prof[dom]
    avg_s = dom_ms * 1e-3 / max(dom_n, 1)
    flops_per_launch = ALGO_FLOPS[dtype] * ncell
    bytes_per_launch = ALGO_WORDS_PATH * es * ncell
    alu_peak = SMS * LANES[dtype] * 2 * sm_max * 1e6 / 1e12      # TFLOP/s
    achieved = flops_per_launch / avg_s / 1e12
    hbm_achieved = bytes_per_launch / avg_s / 1e9
    from paper_1102_5202_b200.binding import fma_peak
    measured_alu = fma_peak("f64" if dtype == "f64" else "f32")   # FMA-chain microbenchmark, after the timed region
    roofline = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s",
                "frac": achieved / alu_peak,
                "traffic": TRAFFIC_BYTES_PER_ZONE[dtype] * ncell,
                "peak_source": f"derived: {SMS} SMs x {LANES[dtype]} {dtype} lanes x 2 x {sm_max:.0f} MHz (DESIGN.md section 5)",
                "algorithmic_flops_per_launch": flops_per_launch, "algorithmic_bytes_per_launch": bytes_per_launch,
                "avg_launch_ms": avg_s * 1e3, "share_of_step": dom_ms / tot_ms if tot_ms > 0 else None,
                "kernels_ms_per_substep": {k: v[0] / (K * SUBSTEPS_PER_STEP) for k, v in prof.items() if v[1]},
                "alu_peak_measured": measured_alu, "frac_of_measured_alu_peak": achieved / measured_alu,
                "hbm_achieved_gbs": hbm_achieved, "hbm_peak_gbs": hbm_gbs, "hbm_frac": hbm_achieved / hbm_gbs,
                "hbm_peak_source": peak_src,
                "traffic_source": "ncu dram bytes of one launch at 128^3, per zone (profiles/r01_substep.md)"}

    # ---- the oracle on the host cores, bounded sample ---------------------------------------------
    cpu = None
    if not args.no_cpu:
        rate, el, cores, _ = oracle_rate(args.ref_n, 1, 1)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{args.ref_n}^3 sub-grid of the same Kerr-Schild sweep, 1 full RK3 step (3 substeps) after "
                         f"1 warm-up step, fp64, {el:.1f} s"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
        "dtype": dtype, "data": "synthetic",
        "config": {"workload": wname,
                   "grid": list(w.n), "substeps_per_step": SUBSTEPS_PER_STEP, "dt": w.dt,
                   "l2": "inputs larger than L2 (resident state %.1f GB)" % (hz.state_bytes / 1e9),
                   "parallelism": ("z-slabs, NCCL halo exchange per substep" if shard else "replicas") if world > 1 else "single"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h_in.numel() * es),
                "d2h_bytes_per_step": int(h_out.numel() * es), "steps": Ke, "ms_per_step": ms_e / Ke},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "cpu_baseline": cpu,
        "state_finite": bool(finite),
        "c2p_fail": d["c2p_fail"], "atm_reset": d["atm_reset"],
        # hz_diagnostics after the timed steps: conservation sums, div B, CFL number
        "diagnostics": {**d, "cfl_number": d["max_speed_over_dx"] * w.dt, "steps_run": W + K},
    }
    print(json.dumps(line))
    hz.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=256, help="cells per axis of the Kerr-Schild sweep")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32", "f32h"],
                    help="f32h = fp32 storage and faces, fp64 flux difference / RK combine / con2prim (PAPER.md:126-128)")
    ap.add_argument("--workload", default="kerr", choices=["kerr", "tube", "alfven", "blast", "tov"],
                    help="which BASELINE.json config to time (default: config 5, the metric's workload)")
    ap.add_argument("--ref-n", type=int, default=128, help="sub-grid the CPU oracle is timed on")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--recon", default="mc", choices=["mc", "ppm"],
                    help="reconstruction (PAPER.md:128): MC-limited linear (the metric's configuration) or PPM")
    ap.add_argument("--shard", action="store_true",
                    help="with --gpus N > 1: cut the one box into N z-slabs with a halo exchange per substep "
                         "(strong scaling) instead of N independent replicas (weak scaling, the default)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
