"""bench.py -- zone-updates/s per RK substep of the HORIZON GRMHD update on B200 (BASELINE.json metric).

Contract: `python bench.py --gpus N --steps K --warmup W [--impl reference]` prints ONE JSON line.

Workload: BASELINE.json config 5, the Kerr-Schild throughput sweep, at 256^3 -- the grid
north_star quotes its target on.  The metric is "fp64 & fp32", so the default run times three legs in one process:
fp64 (the headline `value`; Table 1 reports both precisions), pure fp32 (`"fp32"` object) and
the paper's mixed mode (`"f32h"`: fp32 storage and faces, fp64 flux difference / RK combine / con2prim,
PAPER.md:126-128).  `--dtype f64|f32|f32h` times that one leg only.  A bench "step" is one full third-order
Runge-Kutta step = 3 substeps through `hz_step(dt, 1)`; every substep is one pass of the whole hot path (rows
a1-a9 of DESIGN.md section 2).  `value` = interior cells x 3 x K / device time of the K steps, timed with CUDA
events on the launching stream with per-kernel profiling OFF; the per-kernel split comes from a separate short
profiled pass.  The resident state (46 fields x 134 MB in fp64) is ~50x the 126 MB L2, so every pass streams from
HBM ("inputs larger than L2").

Multi-GPU, one process per GPU: `--gpus N` without torchrun re-executes itself under
`python -m torch.distributed.run`.  Default: N independent replicas (weak scaling, no data-path collective).
`--shard-weak`: ONE box of 256 x 256 x (256 N) cells cut into N z-slabs of 256^3 with a halo exchange per substep
-- the shape of the paper's own weak-scaling run (Table 4).  `--shard`: the one 256^3 box cut into
N slabs (strong scaling).

`--impl reference` times the CPU oracle (oracle/, test infrastructure, as it stands: never tuned) on the host
cores on a bounded sub-grid of the same workload; it is a reported baseline, not the target.
"""
import argparse
import hashlib
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

# Algorithmic words per zone per substep, cleaning on:
# read P(9) + metric(10) + U^(k)(9) + U^n(9, stages 1-2 only -> 6 on average), write U(9) + P(9)
ALGO_WORDS_PATH = 52.0
# ALU peak (B200_PROFILING.md unit counts): 148 SMs x lanes x 2 flop x max SM clock.  The mixed mode runs its
# faces and sources (84 % of its instructions) in fp32 and the rest in fp64: it is rated against the fp32 peak
# and labelled so.
SMS, LANES = 148, {"f64": 64, "f32": 128, "f32h": 128}
ROOFLINE_INPUTS = os.path.join(ROOT, "profiles", "roofline_inputs.json")
KERNEL_SOURCES = ["hz_substep.cuh", "hz_physics.cuh", "hz_kernels.cuh", "hz_layout.cuh", "hz_lib.cu"]


def kernel_source_hash():
    """sha256 over the kernel sources: names the kernel build the ncu-derived roofline inputs belong to."""
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_1102_5202_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def roofline_inputs():
    """Flop numerators and measured DRAM traffic per zone (profiles/roofline_inputs.json: which capture, which
    kernel source they were taken from).  `stale` is set when the kernel sources have changed since."""
    with open(ROOFLINE_INPUTS) as f:
        d = json.load(f)
    d["stale"] = d.get("kernel_source_sha") != kernel_source_hash()
    if d["stale"]:
        print("bench.py: warning: profiles/roofline_inputs.json was taken from another build of the kernels "
              f"({d.get('kernel_source_sha')} != {kernel_source_hash()}); its DRAM traffic figure is out of date",
              file=sys.stderr)
    return d


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

    def window(self, t0, t1):
        """Median SM clock, reasons and peak power of the samples taken between t0 and t1."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for (t, line) in list(self.rows):
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

    def stop(self):
        if self.proc is None:
            return
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()


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
              f"{args.steps} full RK3 steps = {args.steps * 3} substeps, fp64, OpenMP over the outer cell loop; "
              f"the oracle as it stands (plain C++, -O2, never tuned)")
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


def weak_slab_workload(wl, n, rank, world, device):
    """This rank's n^3 slab of the n x n x (n world) Kerr-Schild box (the paper's weak-scaling shape).
    No rank generates the whole box; the one global quantity of the recipe, the maximum of |B| that fixes the
    field's scale, is agreed on with one MAX all-reduce."""
    w = wl.kerr_sweep(n, zmult=world, zslab=(rank * n, (rank + 1) * n))
    g = max_over_ranks(w.extra["bn_max"], world, device)
    w.prim8[5:8] *= w.extra["bn_max"] / g
    return w


def launcher_command(args_list, ngpus, port=None, script=None):
    """The command that runs this file (or `script`) on `ngpus` ranks of one node, one process per GPU: the
    same launch the driver itself uses for N > 1."""
    port = port or int(os.environ.get("MASTER_PORT", "29541"))
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={ngpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), script or os.path.abspath(__file__)] + list(args_list)


def time_leg(args, dtype, w, wname, world, rank, local, barrier, sampler, headline):
    """One timed leg: K full RK3 steps of `w` in `dtype`, device-resident; for the headline leg also the
    end-to-end number through the C ABI with host buffers.  Returns the leg's dictionary."""
    import numpy as np
    import torch
    from paper_1102_5202_b200 import Horizon
    from paper_1102_5202_b200.binding import fma_peak

    K, W = args.steps, max(args.warmup, 3)
    stream = torch.cuda.current_stream()
    es = 8 if dtype == "f64" else 4
    mode = "shard" if (args.shard and world > 1) else ("weak" if (args.shard_weak and world > 1) else "replica")
    dsh = None
    if mode in ("shard", "weak"):
        # z-slabs with ghost planes exchanged over NCCL after every substep (paper_1102_5202_b200/slab.py;
        # PAPER.md:176-178): strong scaling cuts the ONE box, weak scaling gives every rank its own n^3 slab
        from paper_1102_5202_b200 import DistSlabHorizon
        from paper_1102_5202_b200.binding import HZ_HALO_PRIM
        # --exchange fused (default): the neighbours' buffers mapped through CUDA IPC and the exchange done by the
        # substep kernel's own stores (hz_peer_attach); --exchange nccl: pack kernel, NCCL send/recv, unpack kernel
        dsh = DistSlabHorizon(w, dtype=dtype, local=(mode == "weak"), fused=(args.exchange == "fused"))
        hz = dsh.slab.hz
        step = lambda: dsh.step(w.dt, 1)
        ncell = dsh.slab.ncell                                   # this rank's zones
        total_cells = w.ncell if mode == "shard" else world * w.ncell
    else:
        hz = Horizon.from_workload(w, dtype=dtype, stream=stream)
        step = lambda: hz.step(w.dt, 1)
        ncell = w.ncell
        total_cells = world * w.ncell                            # replicas: every rank a full box

    # ---- device-resident timing: inputs in HBM, K x hz_step(dt, 1), profiling off ---------------------------
    for _ in range(W):
        step()
    barrier()
    launches0 = hz.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(stream)
    for _ in range(K):
        step()
    e1.record(stream)
    barrier()
    t1 = time.time()
    ms = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
    launches = hz.launch_count() - launches0
    clocks = sampler.window(t0, t1) if sampler is not None else None
    value = total_cells * SUBSTEPS_PER_STEP * K / (ms * 1e-3)
    # per-kernel split: a separate short pass with hz_profile on (events around every launch)
    hz.profile(True)
    for _ in range(2):
        step()
    prof = hz.profile_read()
    hz.profile(False)
    d = hz.diagnostics() if dsh is None else dsh.diagnostics()
    finite = all(np.isfinite(v) for v in d.values())

    leg = {"dtype": dtype, "value": value, "ms_per_step": ms / K, "gpu_launches": int(launches), "clocks": clocks,
           "state_finite": bool(finite), "c2p_fail": d["c2p_fail"], "atm_reset": d["atm_reset"],
           "c2p_stalled": d["c2p_stalled"], "resident_state_gb": hz.state_bytes / 1e9}

    # ---- end to end through the C ABI with HOST buffers (headline leg) --------------------------------------
    # every step: hz_set_primitives(pinned host prim8) -> hz_step(dt, 1) -> hz_get_primitives(pinned host)
    if headline:
        td = torch.float64 if dtype == "f64" else torch.float32
        h_in = torch.from_numpy(hz.get_primitives()).to(td).pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()
        Ke = max(1, args.e2e_steps if args.e2e_steps > 0 else K)

        def e2e_step():
            hz.set_primitives(h_in)
            if dsh is not None:
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
        ms_e = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
        assert bool(torch.isfinite(h_out).all()), "non-finite primitives after the end-to-end steps"
        leg["e2e"] = {"value": total_cells * SUBSTEPS_PER_STEP * Ke / (ms_e * 1e-3), "unit": UNIT,
                      "h2d_bytes_per_step": int(h_in.numel() * es), "d2h_bytes_per_step": int(h_out.numel() * es),
                      "steps": Ke, "ms_per_step": ms_e / Ke}
        leg["diagnostics"] = {**d, "cfl_number": d["max_speed_over_dx"] * w.dt, "steps_run": W + K + 2 + 2 + Ke}

    # ---- roofline of the dominant kernel ----------------------------------------------
    # The path is bound by plain ALU arithmetic in both precisions (ALU bound 10.1 / 25.7 G zone-updates/s against
    # 15.7 / 31.4 G for HBM), so the roofline is "alu"; the HBM view is reported beside it.
    if rank == 0:
        inp = roofline_inputs()
        hbm_gbs, peak_src, sm_max = peaks()
        tot_ms = sum(v[0] for v in prof.values())
        dom = max(prof, key=lambda k: prof[k][0])
        share = prof[dom][0] / tot_ms if tot_ms > 0 else None
        # average launch duration of the dominant kernel inside the TIMED region: it is the only kernel that
        # launches there (share_of_step from the profiled pass confirms it), 3 K launches in `ms`
        per_sub = (ms / K) / SUBSTEPS_PER_STEP * (share if share else 1.0)
        avg_s = per_sub * 1e-3
        flops = {k: float(v[dtype]) for k, v in inp["flops_per_zone"].items()}
        main = inp["headline_numerator"]
        alu_peak = SMS * LANES[dtype] * 2 * sm_max * 1e6 / 1e12      # TFLOP/s
        achieved = flops[main] * ncell / avg_s / 1e12
        hbm_achieved = ALGO_WORDS_PATH * es * ncell / avg_s / 1e9
        measured_alu = fma_peak("f64" if dtype == "f64" else "f32")  # FMA-chain microbenchmark, after the timed region
        traffic = inp["dram_bytes_per_zone"].get(dtype)
        leg["roofline"] = {
            "bound": "alu", "kernel": dom, "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s",
            "frac": achieved / alu_peak,
            "traffic": traffic * ncell if traffic else None,
            "traffic_source": inp["dram_source"] + (" [STALE: kernels changed since]" if inp["stale"] else ""),
            "peak_source": f"derived: {SMS} SMs x {LANES[dtype]} {'fp32' if dtype != 'f64' else 'fp64'} lanes x 2 x "
                           f"{sm_max:.0f} MHz (DESIGN.md section 5)"
                           + ("; the mixed mode runs phase 2 in fp64, so this fp32 peak is an upper bound of its own"
                              if dtype == "f32h" else ""),
            "flop_numerator": main, "flops_per_zone": flops[main],
            # the same time against every flop count on record (DESIGN.md section 5 says where each comes from)
            "frac_by_numerator": {k: v * ncell / avg_s / 1e12 / alu_peak for k, v in flops.items()},
            "algorithmic_flops_per_launch": flops[main] * ncell,
            "algorithmic_bytes_per_launch": ALGO_WORDS_PATH * es * ncell,
            "avg_launch_ms": avg_s * 1e3, "share_of_step": share,
            "kernels_ms_per_substep": {k: v[0] / (2 * SUBSTEPS_PER_STEP) for k, v in prof.items() if v[1]},
            "alu_peak_measured": measured_alu, "frac_of_measured_alu_peak": achieved / measured_alu,
            "hbm_achieved_gbs": hbm_achieved, "hbm_peak_gbs": hbm_gbs, "hbm_frac": hbm_achieved / hbm_gbs,
            "hbm_peak_source": peak_src, "inputs_kernel_source_sha": inp.get("kernel_source_sha"),
            "inputs_stale": inp["stale"]}
    if dsh is not None:
        dsh.close()
    else:
        hz.close()
    leg["_mode"] = mode
    return leg


def run_gpu(args):
    import dataclasses
    import torch
    import torch.distributed as dist
    import workloads as wl
    from paper_1102_5202_b200 import lib

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

    n = args.n
    if args.shard_weak and world > 1:
        if args.workload != "kerr":
            raise ValueError("--shard-weak stacks Kerr-Schild boxes: use --workload kerr")
        w = weak_slab_workload(wl, n, rank, world, "cuda")
        wname = (f"kerr_sweep {n} x {n} x {n * world}: {world} z-slabs of {n}^3 (BASELINE.json config 5 stacked along z, "
                 f"the paper's weak-scaling shape PAPER.md:244)")
    else:
        w, wname = make_workload(wl, args.workload, n)
    if args.recon == "ppm":
        w = dataclasses.replace(w, params={**w.params, "recon": 1})
        wname += ", PPM reconstruction"

    sampler = None
    if rank == 0:
        sampler = ClockSampler(local)
        sampler.start()
        time.sleep(0.3)
    dtypes = ["f64", "f32", "f32h"] if args.dtype == "all" else [args.dtype]
    legs = [time_leg(args, dt, w, wname, world, rank, local, barrier, sampler, headline=(i == 0))
            for i, dt in enumerate(dtypes)]
    if sampler is not None:
        sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    head = legs[0]
    mode = head.pop("_mode")

    # ---- the oracle on the host cores, bounded sample ---------------------------------------------
    cpu = None
    if not args.no_cpu:
        rate, el, cores, _ = oracle_rate(args.ref_n, 6, 1)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{args.ref_n}^3 sub-grid of the same Kerr-Schild sweep, 6 full RK3 steps (18 substeps) after "
                         f"1 warm-up step, fp64, {el:.1f} s; the unoptimised oracle as it stands (plain C++, -O2)"}

    how = ("halo exchange fused into the substep kernel (stores into the IPC-mapped neighbour), one barrier per substep"
           if args.exchange == "fused" else "NCCL halo exchange per substep")
    par = {"shard": "z-slabs of the one box, " + how, "weak": "one z-slab per rank, " + how, "replica": "replicas"}[mode]
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": head["ms_per_step"], "higher_is_better": True,
        "scaling": "strong" if mode == "shard" else "weak", "vs_baseline": None,
        "dtype": head["dtype"], "data": "synthetic",
        "config": {"workload": wname, "grid": list(w.n), "substeps_per_step": SUBSTEPS_PER_STEP, "dt": w.dt,
                   "l2": "inputs larger than L2 (resident state %.1f GB)" % head["resident_state_gb"],
                   "parallelism": par if world > 1 else "single"},
        "clocks": head["clocks"],
        "e2e": head.get("e2e"),
        "gpu_launches": head["gpu_launches"],
        "roofline": head.get("roofline"),
        "cpu_baseline": cpu,
        "state_finite": head["state_finite"],
        "c2p_fail": head["c2p_fail"], "atm_reset": head["atm_reset"],
        # hz_diagnostics after the timed steps: conservation sums, div B, CFL number
        "diagnostics": head.get("diagnostics"),
    }
    # the other precisions of the metric, measured in the same process after the headline leg
    for leg in legs[1:]:
        leg.pop("_mode")
        key = {"f32": "fp32", "f64": "fp64", "f32h": "f32h"}[leg["dtype"]]
        line[key] = {k: leg[k] for k in ("value", "ms_per_step", "dtype", "gpu_launches", "clocks", "roofline",
                                         "state_finite", "c2p_fail", "atm_reset", "c2p_stalled") if k in leg}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=256, help="cells per axis of the Kerr-Schild sweep")
    ap.add_argument("--dtype", default="all", choices=["all", "f64", "f32", "f32h"],
                    help="all (default): fp64 headline + fp32 and mixed legs; f32h = fp32 storage and faces, fp64 flux "
                         "difference / RK combine / con2prim (PAPER.md:126-128)")
    ap.add_argument("--workload", default="kerr", choices=["kerr", "tube", "alfven", "blast", "tov"],
                    help="which BASELINE.json config to time (default: config 5, the metric's workload)")
    ap.add_argument("--ref-n", type=int, default=128, help="sub-grid the CPU oracle is timed on")
    ap.add_argument("--e2e-steps", type=int, default=0, help="end-to-end steps (0: as many as --steps)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--recon", default="mc", choices=["mc", "ppm"],
                    help="reconstruction (PAPER.md:128): MC-limited linear (the metric's configuration) or PPM")
    ap.add_argument("--shard", action="store_true",
                    help="with --gpus N > 1: cut the one box into N z-slabs with a halo exchange per substep "
                         "(strong scaling) instead of N independent replicas (weak scaling, the default)")
    ap.add_argument("--exchange", default="fused", choices=["fused", "nccl"],
                    help="with --shard / --shard-weak: how the ghost planes travel (fused: peer stores of the substep "
                         "kernel into the CUDA-IPC-mapped neighbour; nccl: pack kernel, send/recv, unpack kernel)")
    ap.add_argument("--shard-weak", action="store_true",
                    help="with --gpus N > 1: one box of n x n x (n N) cells, one n^3 z-slab per rank, halo exchange "
                         "per substep (weak scaling in the paper's own shape, PAPER.md:244)")
    args = ap.parse_args(argv)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the N ranks ourselves (one process per GPU) and hand back their exit code
        return subprocess.call(launcher_command(sys.argv[1:] if argv is None else argv, args.gpus))
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
