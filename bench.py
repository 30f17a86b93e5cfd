#!/usr/bin/env python
"""bench.py — headline benchmark of the B200 metadynamics hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config c3] [--precision 32|64]

A "step" = one pass of the whole hot path (neighbour build -> CVs -> bias -> forces -> deposit) over
one synthetic system.  Default workload: BASELINE.json configs[3] (1,024,000-atom GaN-shaped Q6 step,
10,000 well-tempered hills), the configuration the metric "atom-steps/s at 1M atoms" is quoted on.
Prints ONE JSON line (rank 0).  Multi-GPU: the path does not shard ("replicas only");
--gpus N runs N independent replicas, one process per GPU, weak scaling, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "CV+bias+force atom-steps/s at 1M atoms"
UNIT = "atom-steps/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c3", choices=["c0", "c1", "c2", "c3", "c4", "t0", "g0", "r0"])
    ap.add_argument("--precision", type=int, default=0, help="0 = the workload's own (c3: 32 for the headline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fast-setup", action="store_true",
                    help="profiling runs only: seeded hill heights instead of the well-tempered replay, no e2e leg")
    ap.add_argument("--lazy", action="store_true", help="params.lazy_neighbors: skip the list build when no CV reads it (c1, t0)")
    ap.add_argument("--virial", action="store_true", help="also compute the bias virial every step (NPT; COORD / Q6 / LATTICE CVs)")
    ap.add_argument("--stage-times", action="store_true", default=True)
    ap.add_argument("--skin", type=float, default=0.0,
                    help="params.skin: Verlet-skin reuse of the neighbour list (a separately reported mode; the headline rebuilds "
                         "the list every step)")
    ap.add_argument("--move", type=float, default=0.0,
                    help="move every atom by a seeded Gaussian displacement of this width (A) before every timed step (device "
                         "kernels of the harness, outside the timed events): what an MD integrator does between two calls")
    ap.add_argument("--decompose", action="store_true",
                    help="slab decomposition of ONE c3 / c4 system over the ranks (strong scaling; DESIGN.md section 8): halo of "
                         "2 (rc + skin), one all-reduce of ncv doubles per step.  Default without it: N independent replicas")
    ap.add_argument("--as-rank", type=int, default=-1,
                    help="with --decompose on ONE GPU: time the share of this rank of a world of --of ranks alone (no all-reduce)")
    ap.add_argument("--of", type=int, default=1)
    ap.add_argument("--peaks", action="store_true",
                    help="only measure the scalar-pipe roofline denominators (FP32 / FP32x2 / FP64 FMA microbenchmark, "
                         "metad_fma_peak) and print them as one JSON line")
    return ap.parse_args()


def workload(name):
    from paper_2510_06873_b200.inputs import configs
    return configs.BUILDERS[name]()


def describe(w, precision):
    kinds = {0: "coordination", 1: "Q6 mean", 2: "Q6 solid-like count", 3: "radius of gyration", 4: "native contacts", 5: "torsion", 6: "distance to nearest", 7: "lattice parameter"}
    wl = {"t0": "PAPER.md:37 alanine-dipeptide-shaped torsion workload (t0, SURVEY.md §8(f) NEXT-1)",
          "r0": "PAPER.md:43 surface-O ... nearest-H distance, well-tempered, on the configs[2] slab + water structure (r0)",
          "g0": "PAPER.md:51 GaN CV set (coordination number + 3 lattice parameters) on the configs[3] structure (g0)"
          }.get(w.name, f"BASELINE.json configs[{w.name[1]}] ({w.name})")
    return {"workload": wl, "atoms": int(w.natoms),
            "cvs": [kinds[c.kind] for c in w.cvs], "hills": int(w.n_hills), "rc": w.rc,
            "pair_precision": f"fp{precision}", "stride": int(w.stride), "virial": bool(getattr(w, "_virial", False)),
            "neighbour_build": ("skipped (lazy_neighbors: no CV of this workload reads the list)"
                                if (w.name in ("t0", "r0") or getattr(w, "_lazy", False)) and all(c.kind in (3, 4, 5, 6, 7) for c in w.cvs)
                                else "every step, list-free (lazy_neighbors: the candidate scan accumulates the coordination sum and "
                                     "the per-atom gradient and stores no list)"
                                if getattr(w, "_lazy", False) and precision == 32 and not getattr(w, "_virial", False)
                                and w.max_neigh <= 32 and any(c.kind == 0 and c.group_a is None and c.group_b is None for c in w.cvs)
                                and not any(c.kind in (1, 2, 6) for c in w.cvs)
                                else "every step"),
            "l2": ("per-step working set (neighbour list + q6 records + positions + forces) exceeds the 126 MB L2; no flush"
                   if w.natoms * (4 * w.max_neigh + 64 + 16 + 24 + 16) > 126e6 else
                   "working set fits the 126 MB L2 and is not flushed: this workload is bound by the latency of its ~10 "
                   "dependent kernel launches per step, not by memory")}


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_sample(name, full=False):
    """A bounded sample of the workload for the CPU oracle (same recipe, fewer atoms)."""
    from paper_2510_06873_b200.inputs import configs
    if name == "c3" and full:
        return configs.config3(), "none: the full BASELINE.json configs[3] workload (1,024,000 atoms, 10,000 hills), one step"
    if name == "c3":
        return configs.config3(cells=(30, 30, 16), sphere_r=18.0, n_hills=10000), "c3 recipe at 30x30x16 cells (57,600 atoms), 10,000 hills"
    if name == "c4":
        return configs.config4(cells=(30, 30, 16), sphere_r=18.0, n_hills=20000, grid=(0, 0)), "c4 recipe at 57,600 atoms, 20,000 hills, exact sum"
    if name == "g0":
        return configs.config_g0(cells=(30, 30, 16), sphere_r=18.0, n_hills=10000), "g0 recipe at 30x30x16 cells (57,600 atoms), 10,000 hills"
    w = configs.BUILDERS[name]()
    return w, f"{name} at full size"


def oracle_time_steps(w, nsteps):
    """Times the oracle as it stands (never tuned) on the host cores: full steps incl. neighbour build."""
    import oracle
    from oracle.reference import OracleMetaD
    from paper_2510_06873_b200.inputs import hill_walk, hill_walk_periodic, seeded_heights
    o = OracleMetaD(w)
    o.build_neighbors(w.pos)
    s0 = o.eval_cv(want_grad=False)
    if w.hill_centers is not None:
        o.set_hills(w.hill_centers, w.hill_heights)
    elif w.period:
        o.set_hills(hill_walk_periodic(5, s0, w.sigma, w.n_hills, w.period, w.extra["period_lo"]),
                    seeded_heights(5, w.n_hills, w.w0))
    else:
        o.set_hills(hill_walk(5, s0, w.sigma, w.n_hills), seeded_heights(5, w.n_hills, w.w0))
    F = np.zeros((w.natoms, 3))
    times = []
    for _ in range(nsteps):
        t = time.perf_counter()
        o.run_step(w.pos, F)
        times.append(time.perf_counter() - t)
    return times, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, desc = oracle_sample(args.config)
    steps = max(1, min(args.steps, 5))
    warm = 1 if args.warmup > 0 else 0
    times, cores = oracle_time_steps(w, warm + steps)
    times = times[warm:]
    total = sum(times)
    value = w.natoms * len(times) / total
    full = workload(args.config) if args.config in ("c0", "c1", "c2") else None
    cfg = describe(w if full is None else full, 64)
    if args.config in ("c3", "c4"):
        cfg["workload"] = f"BASELINE.json configs[{args.config[1]}] ({args.config})"
    cfg["sample"] = desc
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": len(times),
            "warmup": warm, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ multi-process plumbing
def max_over_ranks(values, device="cuda"):
    """Element-wise max over all ranks of a list of floats (device-timed durations): the whole job is
    as slow as its slowest replica.  Works with NCCL (cuda tensors) and gloo (cpu tensors)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def job_throughput(world, atoms_per_replica, steps, ms_max):
    """Replicas only: N independent copies of the workload, value = all atoms x steps / slowest time."""
    return world * atoms_per_replica * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------ our arm
def prepare_hills(w, md_cls, precision, dpos, torch):
    """Hill centres = seeded walk around the structure's own CV (reading K); heights by replaying the
    well-tempered rule through the library's own bias+deposit kernels (stride-1 helper context)."""
    from paper_2510_06873_b200.inputs import hill_walk, hill_walk_periodic
    import copy
    if w.hill_centers is not None:
        return np.asarray(w.hill_centers), np.asarray(w.hill_heights)
    probe = md_cls(w, precision=precision, max_hills=8)
    probe.build_neighbors(dpos)
    probe.eval_cv()
    probe.synchronize()
    s0 = probe.cv.cpu().numpy()
    probe.close()
    if w.period:
        centers = hill_walk_periodic(5, s0, w.sigma, w.n_hills, w.period, w.extra["period_lo"])
    else:
        centers = hill_walk(5, s0, w.sigma, w.n_hills)
    w1 = copy.copy(w)
    w1.stride = 1
    w1.cvs = w.cvs
    rep = md_cls(w1, precision=precision, max_hills=w.n_hills + 8)
    with torch.cuda.stream(rep.stream):
        dc = torch.tensor(centers, device="cuda")
    rep.synchronize()
    for k in range(w.n_hills):
        rep.bias(cv=dc[k])
        rep.deposit(cv=dc[k])
    c, h = rep.get_hills()
    rep.close()
    return c, h


# Algorithmic (compulsory) work per atom, DESIGN.md §6.  nb = mean neighbours, T = bytes per scalar.
def algo_q6_force_bytes(nb, T):
    # neighbour entries 4*nb + count 4, own position 4*T, q6 records 16*T (each read once), perm 4, force read+write 6*T
    return 4 * nb + 4 + 4 * T + 16 * T + 4 + 6 * T


def algo_build_flops(nb, cand=94.5):
    # candidate scan: 3 sub + (1 mul + 2 fma = 5 flop) + 1 compare = 9 flop per candidate (9 rows x 2.5 cells x 4.2 atoms = 94.5);
    # fused Q6 pass 1 per neighbour: r2 5, rsqrt 1, unit vector 3, E polynomials 20, (x+iy)^m recurrence 30, 13 fma = 26 -> 85
    return 9.0 * cand + 85.0 * nb


def algo_coord_build_flops(nb, cand=94.5):
    # candidate scan as above; per neighbour on the exact pass: r2 5, sqrt 1, x = r / r0 1, x^5 and x^6 5, 1 / (1 + x^6) 2,
    # sw' 3, sum 1, rsqrt 1, pair factor 3, three fma 6 -> 28
    return 9.0 * cand + 28.0 * nb


FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # nominal FMA peak from the guide's unit counts and clocks
FP64_NOMINAL_TFLOPS = FP32_NOMINAL_TFLOPS / 2            # B200: one FP64 FMA lane per two FP32 lanes
ISSUE_PEAK_GINST = 148 * 4 * 1.965                      # warp instructions / ns


def algo_q6_force_flops(nb):
    # per pair: 13 fma for the combined record 26, d and r 9, rsqrt + unit vector 5, Y6m (E polynomials 20, recurrence 30),
    # gradient (6 x 14 + 8) 92, tangent projection and 1/r 14, sum 3 -> ~199; per atom: own record 13, force update 9
    return 199.0 * nb + 22.0


def algo_grid_build_flops(nodes, hills):
    # separable tile build (bias.cu: k_grid_accumulate): per node and hill g = ex ey, v += g, v0 += g ga, v1 += g gb,
    # v01 += (g ga) gb = 9 flop; the 1-D factors (one exp per hill and tile row / column) add 2 x 16 exps per 256 node-hills
    return 9.0 * nodes * hills


def measure_peaks():
    """Scalar-pipe roofline denominators, measured on this GPU right now."""
    from paper_2510_06873_b200 import metad
    out = {}
    for kind in ("f32", "f32x2", "f64"):
        tf, ms = metad.fma_peak(kind)
        out[kind] = {"tflops": tf, "ms": ms}
    out["nominal"] = {"f32": FP32_NOMINAL_TFLOPS, "f64": FP64_NOMINAL_TFLOPS}
    out["how"] = ("metad_fma_peak: 8 dependent-free FMA chains per thread, 2,048 threads per SM on every SM, CUDA events, best of 4 "
                  "launches after 2 warm-up launches")
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2510_06873_b200.metad import MetaD

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w = workload(args.config)
    w._virial = bool(args.virial)
    w._lazy = bool(args.lazy)
    precision = args.precision or (32 if args.config in ("c3", "c4", "g0") else w.precision)
    tdt = torch.float32 if precision == 32 else torch.float64
    pos = w.pos.astype(np.float32 if precision == 32 else np.float64)
    dpos = torch.tensor(pos, device="cuda")
    torch.cuda.synchronize()
    if args.fast_setup:
        from paper_2510_06873_b200.inputs import hill_walk, seeded_heights
        if w.period:
            from paper_2510_06873_b200.inputs import hill_walk_periodic
            centers = hill_walk_periodic(5, np.zeros(w.ncv), w.sigma, w.n_hills, w.period, w.extra["period_lo"])
        else:
            centers = hill_walk(5, np.full(w.ncv, 0.23), w.sigma, w.n_hills)
        heights = seeded_heights(5, w.n_hills, w.w0)
    else:
        centers, heights = prepare_hills(w, MetaD, precision, dpos, torch)

    grid = None
    if w.grid_n[0] and w.period:
        lo = np.asarray(w.extra["period_lo"], dtype=np.float64)
        grid = (w.grid_n, lo, lo + np.asarray(w.period))                        # reading X: one period
    elif w.grid_n[0]:
        sig = np.asarray(w.sigma)
        grid = (w.grid_n, centers[0] - 120 * sig, centers[0] + 120 * sig)      # reading M
    md = MetaD(w, precision=precision, max_hills=w.n_hills + args.steps + args.warmup + 4096, grid=grid,
               want_virial=args.virial, lazy_neighbors=(args.config in ("t0", "r0") or args.lazy), skin=args.skin)
    md.set_hills(centers, heights)
    with torch.cuda.stream(md.stream):
        F = torch.zeros((w.natoms, 3), device="cuda", dtype=tdt)
    md.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timed region: K graph replays
    moving = args.move > 0.0
    if moving:
        # the harness plays the MD integrator: seeded Gaussian displacement + re-wrapping into the (triclinic) box, on the
        # context's stream, OUTSIDE the timed events; the library sees new coordinates in the same device buffer every step
        gen = torch.Generator(device="cuda")
        gen.manual_seed(2510068730 + rank)
        Bm = torch.tensor(w.box.reshape(3, 3), device="cuda", dtype=torch.float64)
        Binv = torch.linalg.inv(Bm)

        def integrate():
            with torch.cuda.stream(md.stream):
                dpos.add_(torch.randn(dpos.shape, device="cuda", dtype=dpos.dtype, generator=gen) * args.move)
                fr = dpos.double() @ Binv
                fr -= torch.floor(fr)
                dpos.copy_((fr @ Bm).to(dpos.dtype))
    for _ in range(args.warmup):
        if moving:
            integrate()
        md.run(dpos, F, 1)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = md.launch_count()
    b0 = md.rebuilds()
    if moving:
        evs_ = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a_, b_ in evs_:
            integrate()
            a_.record(md.stream)
            md.run(dpos, F, 1)
            b_.record(md.stream)
        barrier()
        ms = float(sum(a_.elapsed_time(b_) for a_, b_ in evs_))
    else:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(md.stream)
        md.run(dpos, F, args.steps)
        e1.record(md.stream)
        barrier()
        ms = e0.elapsed_time(e1)
    launches = md.launch_count() - l0
    builds = md.rebuilds() - b0
    # ---- per-stage CUDA-event times (same stream, explicit five calls), inside the same clock-sampled window
    stage_names = ["build_neighbors", "eval_cv", "bias", "apply_forces", "deposit"]
    acc = np.zeros(5)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
    reps = max(3, min(args.steps, 20))
    for it in range(reps + 2):
        evs[0].record(md.stream)
        md.build_neighbors(dpos); evs[1].record(md.stream)
        md.eval_cv(); evs[2].record(md.stream)
        md.bias(); evs[3].record(md.stream)
        md.apply_forces(F); evs[4].record(md.stream)
        md.deposit(); evs[5].record(md.stream)
        md.synchronize()
        if it >= 2:
            acc += np.array([evs[k].elapsed_time(evs[k + 1]) for k in range(5)])
    stage_ms = acc / reps
    sort_ms = list_ms = None
    try:
        md.set_timing(True)
        ts = []
        for it in range(5):
            md.build_neighbors(dpos)
            ts.append(md.get_timing())
        md.set_timing(False)
        sort_ms, list_ms = float(np.median([t[0] for t in ts[1:]])), float(np.median([t[1] for t in ts[1:]]))
    except Exception:
        pass
    clocks = sampler.stop() if rank == 0 else None
    status = md.status()
    state = md.state()

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    # host buffers from the library's own page-locked allocator (include/metad.h: metad_host_alloc)
    from paper_2510_06873_b200.metad import pinned_array
    pos_h = pinned_array(pos.shape, pos.dtype)
    pos_h[...] = pos
    F_h = pinned_array((w.natoms, 3), pos.dtype)
    F_h[...] = 0
    for _ in range(min(args.warmup, 3)):
        md.step_host(pos_h, F_h)
    barrier()
    ke = 1 if args.fast_setup else max(3, min(args.steps, 20))
    t0 = time.perf_counter()
    for _ in range(ke):
        md.step_host(pos_h, F_h)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0

    ms_max, e2e_ms_max = max_over_ranks([ms, e2e_s * 1e3])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = job_throughput(world, w.natoms, args.steps, ms_max)
    e2e_value = job_throughput(world, w.natoms, ke, e2e_ms_max)
    tb = 4 if precision == 32 else 8
    peaks = {}
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        peaks = json.load(open(pk))
    hbm_peak, peak_src = (peaks["hbm_gbs"], "measured (MEASURED_PEAKS.json hbm_gbs)") if "hbm_gbs" in peaks else (6650.0, "fallback (B200_PROFILING.md)")
    fpk = measure_peaks()
    f32_peak, f64_peak = fpk["f32"]["tflops"], fpk["f64"]["tflops"]
    f32_src = f"measured: metad_fma_peak FP32 FFMA {f32_peak:.1f} TFLOP/s (nominal 148 x 128 x 2 x 1.965 GHz = {FP32_NOMINAL_TFLOPS:.1f})"
    f64_src = f"measured: metad_fma_peak FP64 DFMA {f64_peak:.1f} TFLOP/s (nominal {FP64_NOMINAL_TFLOPS:.1f})"
    roof, roof_all = None, []
    traffic = {}
    tpath = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get(f"{args.config}_fp{precision}", {})
    if any(c.kind in (1, 2) for c in w.cvs):
        cnt, _ = md.neighbors()
        nb = float(cnt.mean())
        # a6: the gather-form force kernel against the HBM roofline (north_star: "HBM GB/s ... for the force pass")
        bytes_launch = algo_q6_force_bytes(nb, tb) * w.natoms
        ach = bytes_launch / (stage_ms[3] * 1e-3) / 1e9
        kname = "k_q6_force_g" if precision == 32 else "k_q6_force<double>"
        r_force = {"kernel": f"{kname} (stage apply_forces)", "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s",
                   "frac": ach / hbm_peak, "traffic": traffic.get("force_dram_bytes"), "peak_source": peak_src,
                   "algorithmic_bytes_per_launch": bytes_launch, "kernel_ms": float(stage_ms[3]), "mean_neighbours": nb}
        roof_all.append(r_force)
        roof = r_force
        # the same kernel against the scalar pipe it computes on (north_star: "FP32/FP64 pipe utilisation for the Q6 ... passes")
        ffl = algo_q6_force_flops(nb) * w.natoms
        pk_, src_ = (f32_peak, f32_src) if precision == 32 else (f64_peak, f64_src)
        roof_all.append({"kernel": f"{kname} (stage apply_forces), scalar-pipe view", "bound": "alu",
                         "achieved": ffl / (stage_ms[3] * 1e-3) / 1e12, "peak": pk_, "unit": "TFLOP/s",
                         "frac": ffl / (stage_ms[3] * 1e-3) / 1e12 / pk_, "traffic": traffic.get("force_dram_bytes"),
                         "peak_source": src_, "algorithmic_flops_per_launch": ffl, "kernel_ms": float(stage_ms[3])})
        if precision == 64 and list_ms is not None and stage_ms[1] < 0.25 * list_ms:
            # tiled fp64 path (csrc/tiled64.cu): the list build fused with Q6 pass 1 in fp64 pair math; eval_cv only hands the
            # sums over.  Same algorithmic count as the fp32 build, against the measured FP64 pipe
            fl = algo_build_flops(nb) * w.natoms
            ach_tf = fl / (list_ms * 1e-3) / 1e12
            roof_all.append({"kernel": "k_tile_build64 (list phase of build_neighbors)", "bound": "alu", "achieved": ach_tf,
                             "peak": f64_peak, "unit": "TFLOP/s", "frac": ach_tf / f64_peak, "traffic": traffic.get("build_dram_bytes"),
                             "peak_source": f64_src, "algorithmic_flops_per_launch": fl, "kernel_ms": float(list_ms),
                             "sort_phase_ms": float(sort_ms)})
            if list_ms > stage_ms[3]:
                roof = roof_all[-1]                # the dominant kernel of the fp64 step
        elif precision == 64:
            # generic fp64 path: list build and Q6 pass 1 are separate kernels (stage times), both on the FP64 pipe
            p1 = (85.0 * nb) * w.natoms
            roof_all.append({"kernel": "k_q6_pass1<double> (stage eval_cv)", "bound": "alu",
                             "achieved": p1 / (stage_ms[1] * 1e-3) / 1e12, "peak": f64_peak, "unit": "TFLOP/s",
                             "frac": p1 / (stage_ms[1] * 1e-3) / 1e12 / f64_peak, "traffic": None, "peak_source": f64_src,
                             "algorithmic_flops_per_launch": p1, "kernel_ms": float(stage_ms[1])})
        if precision == 32 and args.skin > 0.0:
            # skin mode: the stage calls above found the list still valid, so eval_cv timed k_q6_pass1_g (Q6 pass 1 over the stored
            # rc + skin list).  Algorithmic bytes: the list entries (4 B each, mean rc + skin count), the sorted positions once,
            # the 64-byte record and q6 / f' written per atom; flops: the same Y6m accumulation as the fused build (85 per pair)
            nbl = nb * ((w.rc + args.skin) / w.rc) ** 3
            by1 = (4.0 * nbl + 16 + 64 + 8 + 4.0 * nb) * w.natoms
            a1 = by1 / (stage_ms[1] * 1e-3) / 1e9
            roof_all.append({"kernel": "k_q6_pass1_g (stage eval_cv, list kept)", "bound": "hbm", "achieved": a1, "peak": hbm_peak,
                             "unit": "GB/s", "frac": a1 / hbm_peak, "traffic": None, "peak_source": peak_src,
                             "algorithmic_bytes_per_launch": by1, "kernel_ms": float(stage_ms[1]), "mean_list_entries": nbl})
            if stage_ms[1] > stage_ms[3]:
                roof = roof_all[-1]                # the dominant kernel of a step that keeps its list
            fl1 = (12.0 * nbl + 85.0 * nb) * w.natoms
            roof_all.append({"kernel": "k_q6_pass1_g, scalar-pipe view", "bound": "alu", "achieved": fl1 / (stage_ms[1] * 1e-3) / 1e12,
                             "peak": f32_peak, "unit": "TFLOP/s", "frac": fl1 / (stage_ms[1] * 1e-3) / 1e12 / f32_peak,
                             "traffic": None, "peak_source": f32_src, "algorithmic_flops_per_launch": fl1,
                             "kernel_ms": float(stage_ms[1])})
        elif precision == 32 and list_ms is not None:
            # a1+a3: candidate scan fused with Q6 pass 1 — plain FP32 ALU / issue bound (no tensor-core work on this path)
            fl = algo_build_flops(nb) * w.natoms
            ach_tf = fl / (list_ms * 1e-3) / 1e12
            r_build = {"kernel": "k_tile_build<Q6> (list phase of build_neighbors)", "bound": "alu", "achieved": ach_tf,
                       "peak": f32_peak, "unit": "TFLOP/s", "frac": ach_tf / f32_peak,
                       "traffic": traffic.get("build_dram_bytes"), "peak_source": f32_src,
                       "algorithmic_flops_per_launch": fl, "kernel_ms": float(list_ms), "sort_phase_ms": float(sort_ms)}
            roof_all.append(r_build)
            if list_ms > stage_ms[3]:
                roof = r_build                     # the dominant kernel of the step
            # what actually binds both kernels is instruction issue (profiles/r2i_ncu.md), so the same launches are also put
            # against the issue peak 148 SMs x 4 schedulers x 1.965 GHz, with the executed warp instructions ncu counted
            for key, kms, nm in (("build_warp_instructions", list_ms, "k_tile_build<Q6>"), ("force_warp_instructions", stage_ms[3], "k_q6_force_g")):
                if traffic.get(key):
                    gi_ = traffic[key] / (kms * 1e-3) / 1e9
                    roof_all.append({"kernel": f"{nm}, issue-slot view", "bound": "alu", "achieved": gi_, "peak": ISSUE_PEAK_GINST,
                                     "unit": "G warp-instructions/s", "frac": gi_ / ISSUE_PEAK_GINST, "traffic": None,
                                     "peak_source": "148 SMs x 4 schedulers x 1.965 GHz (guide's unit counts); instruction count from "
                                                    "profiles/ncu_traffic.json (ncu smsp__inst_executed.sum of the same kernel)",
                                     "warp_instructions_per_launch": traffic[key], "kernel_ms": float(kms)})
    elif (precision == 32 and list_ms is not None and not args.virial and not args.lazy
          and sum(c.kind == 0 and c.group_a is None and c.group_b is None for c in w.cvs) == 1
          and getattr(w, "max_neigh", 64) <= 32):
        # tiled coordination path (g0): the list build with the sum of sw and its per-atom gradient riding on the exact pass
        # is the dominant kernel (the force stage is one scaled add per atom) — FP32 ALU / issue bound like the Q6 build
        cnt, _ = md.neighbors()
        nb = float(cnt.mean())
        fl = algo_coord_build_flops(nb) * w.natoms
        ach_tf = fl / (list_ms * 1e-3) / 1e12
        roof = {"kernel": "k_tile_build<coordination> (list phase of build_neighbors)", "bound": "alu", "achieved": ach_tf,
                "peak": f32_peak, "unit": "TFLOP/s", "frac": ach_tf / f32_peak,
                "traffic": traffic.get("build_dram_bytes"), "peak_source": f32_src,
                "algorithmic_flops_per_launch": fl, "kernel_ms": float(list_ms), "sort_phase_ms": float(sort_ms),
                "mean_neighbours": nb}
        roof_all.append(roof)
    lps = int(launches) // max(args.steps, 1)
    if roof is None:
        # c0-c2, t0, r0: a handful of dependent launches of a few microseconds each in one CUDA graph.  The dominant stage is
        # reported against HBM with its compulsory bytes, and the line says what really bounds it: launch latency.
        k = int(np.argmax(stage_ms))
        nbm = 0.0
        try:
            cnt, _ = md.neighbors()
            nbm = float(cnt.mean())
        except Exception:
            pass                                        # lazy_neighbors: no list in this context
        by = w.natoms * ((3 * tb + 2 * 4 * tb + 4 * nbm + 8) if k == 0 else 3 * tb)
        ach = by / (stage_ms[k] * 1e-3) / 1e9
        roof = {"kernel": f"stage {stage_names[k]} (generic kernels)", "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s",
                "frac": ach / hbm_peak, "traffic": None, "peak_source": peak_src, "algorithmic_bytes_per_launch": by,
                "kernel_ms": float(stage_ms[k]), "mean_neighbours": nbm, "launch_bound": True, "launches_per_step": lps,
                "us_per_launch": 1e3 * ms_max / args.steps / max(lps, 1),
                "note": "latency-bound: the step is a chain of dependent launches of 2-10 us each; neither HBM nor the ALUs are near a roof"}
        roof_all.append(roof)
    if grid is not None:
        # a5g: time of the table build over all hills (metad_set_hills: separable 16 x 16-node tiles), FP64 pipe
        g0_, g1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        md.synchronize()
        nh_now = md.state()["nhills"]
        ch, hh = md.get_hills()
        g0_.record(md.stream)
        md.set_hills(ch, hh)
        g1_.record(md.stream)
        torch.cuda.synchronize()
        gms = g0_.elapsed_time(g1_)
        gfl = algo_grid_build_flops(grid[0][0] * grid[0][1], nh_now)
        roof_all.append({"kernel": "k_grid_accumulate (metad_set_hills: whole-table build, not a per-step kernel)", "bound": "alu",
                         "achieved": gfl / (gms * 1e-3) / 1e12, "peak": f64_peak, "unit": "TFLOP/s",
                         "frac": gfl / (gms * 1e-3) / 1e12 / f64_peak, "traffic": None, "peak_source": f64_src,
                         "algorithmic_flops_per_launch": gfl, "kernel_ms": float(gms), "hills": int(nh_now),
                         "nodes": [int(grid[0][0]), int(grid[0][1])],
                         "gaussian_terms_per_s": grid[0][0] * grid[0][1] * nh_now / (gms * 1e-3)})
    cfg_ = describe(w, precision)
    if args.skin > 0.0:
        cfg_["neighbour_build"] = (f"Verlet skin {args.skin} A (params.skin): the rc + skin list is kept while no atom has moved "
                                   f"{args.skin / 2} A; {int(builds)} builds in {args.steps} timed steps, decided on the device")
    cfg_["positions"] = (f"moved before every step by a seeded Gaussian displacement of width {args.move} A and re-wrapped (harness "
                         "kernels outside the timed events)" if moving else "fixed (BASELINE.json configs: evaluate with fixed positions)")
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if precision == 32 else "f64", "data": "synthetic", "config": cfg_,
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(pos_h.nbytes + F_h.nbytes),
                    "d2h_bytes_per_step": int(F_h.nbytes + 8 * (w.ncv + 1)), "ms_per_step": e2e_ms_max / ke},
            "roofline": roof, "roofline_kernels": roof_all, "peaks": fpk, "graph": md.graph_info(),
            "list_builds_in_timed_steps": int(builds),
            "stages_ms": {n: float(v) for n, v in zip(stage_names, stage_ms)},
            "state": {"cv": [float(x) for x in state["cv"]], "V": float(state["V"]), "nhills": state["nhills"],
                      "sticky": status}}
    if w.period and w.ncv == 2:
        # NEXT-2: reweighting of a synthetic 2^20-frame CV trajectory against the workload's hills
        from paper_2510_06873_b200.inputs import hill_walk_periodic
        T = 1 << 20
        traj = hill_walk_periodic(9, np.zeros(2), [1.0, 1.0], T, w.period, w.extra["period_lo"], step_frac=0.3)
        with torch.cuda.stream(md.stream):
            dt = torch.tensor(traj, device="cuda")
        md.synchronize()
        lo = np.asarray(w.extra["period_lo"]); hi = lo + np.asarray(w.period)
        md.reweight(dt, (128, 128), lo, hi)
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record(md.stream)
        Pm, Fm = md.reweight(dt, (128, 128), lo, hi)
        r1.record(md.stream)
        torch.cuda.synchronize()
        rms = r0.elapsed_time(r1)
        nh = md.state()["nhills"]
        line["reweight"] = {"frames": T, "hills": int(nh), "bins": [128, 128], "ms": rms,
                            "gaussian_evals_per_s": T * nh / (rms * 1e-3), "dtype": "f64",
                            "fes_span_kT": float((Fm[np.isfinite(Fm)].max() - Fm.min()) / w.kT)}
    if not args.no_cpu_baseline and world == 1:
        ws, desc = oracle_sample(args.config, full=True)
        times, cores = oracle_time_steps(ws, 1 if ws.natoms > 500000 else 2)
        line["cpu_baseline"] = {"value": ws.natoms / times[-1], "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": desc, "s_per_step": times[-1]}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_decomposed(args):
    """--decompose: ONE system cut into slabs along c, one rank per GPU (paper_2510_06873_b200/domain.py).  Stage calls +
    metad_cv_owned_sum + an all-reduce of ncv doubles per step; value = atoms of the WHOLE system x steps / slowest rank."""
    import torch
    import torch.distributed as dist
    from paper_2510_06873_b200 import domain
    from paper_2510_06873_b200.inputs import hill_walk, seeded_heights
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.config not in ("c3", "c4"):
        raise SystemExit("--decompose: the Q6 workloads c3 and c4 (DESIGN.md section 8)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    solo = args.as_rank >= 0                       # one rank's share, alone on this GPU
    dworld, drank = (args.of, args.as_rank) if solo else (world, rank)
    w = workload(args.config)                      # every rank builds the same seeded system
    precision = args.precision or 32
    tdt = torch.float32 if precision == 32 else torch.float64
    centers, heights = hill_walk(5, np.full(w.ncv, 0.23), w.sigma, w.n_hills), seeded_heights(5, w.n_hills, w.w0)
    rk = domain.SlabMetaD(w, dworld, drank, precision=precision, skin=args.skin, max_hills=w.n_hills + args.steps + args.warmup + 64)
    md = rk.md
    md.set_hills(centers, heights)
    nloc = len(rk.local)
    pos_h = torch.tensor(w.pos[rk.local].astype(np.float32 if precision == 32 else np.float64)).pin_memory()
    F_h = torch.zeros((nloc, 3), dtype=tdt).pin_memory()
    with torch.cuda.stream(md.stream):
        dpos = pos_h.to("cuda", non_blocking=True)
        F = torch.zeros((nloc, 3), device="cuda", dtype=tdt)
    md.synchronize()

    def step():
        rk.phase1(dpos)
        if not solo:
            rk.all_reduce()
        rk.phase2(F)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = md.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(md.stream)
    for _ in range(args.steps):
        step()
    e1.record(md.stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = md.launch_count() - l0
    # stage times of this rank
    names = ["build_neighbors", "eval_cv", "cv_owned_sum", "all_reduce", "bias", "apply_forces", "deposit"]
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(8)]
    acc = np.zeros(7)
    for it in range(7):
        evs[0].record(md.stream)
        md.build_neighbors(dpos); evs[1].record(md.stream)
        md.eval_cv(); evs[2].record(md.stream)
        md.cv_owned_sum(rk.d_owned); evs[3].record(md.stream)
        if not solo:
            rk.all_reduce()
        evs[4].record(md.stream)
        md.bias(); evs[5].record(md.stream)
        md.apply_forces(F); evs[6].record(md.stream)
        md.deposit(); evs[7].record(md.stream)
        barrier()
        if it >= 2:
            acc += np.array([evs[k].elapsed_time(evs[k + 1]) for k in range(7)])
    stage_ms = acc / 5
    clocks = sampler.stop() if rank == 0 else None
    # end to end: this rank's positions and forces from / to page-locked host memory inside the timed region
    ke = max(3, min(args.steps, 20))
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        with torch.cuda.stream(md.stream):
            dpos.copy_(pos_h, non_blocking=True)
            F.copy_(F_h, non_blocking=True)
        step()
        with torch.cuda.stream(md.stream):
            F_h.copy_(F, non_blocking=True)
            cv_h = md.cv.cpu()
        md.synchronize()
    e2e_s = time.perf_counter() - t0
    ms_max, e2e_ms_max = max_over_ranks([ms, e2e_s * 1e3])
    status = md.status()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    natoms_job = w.natoms                           # strong scaling: the whole system, whatever the number of ranks
    value = natoms_job * args.steps / (ms_max * 1e-3)
    tb = 4 if precision == 32 else 8
    peaks = {}
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        peaks = json.load(open(pk))
    hbm_peak, peak_src = (peaks["hbm_gbs"], "measured (MEASURED_PEAKS.json hbm_gbs)") if "hbm_gbs" in peaks else (6650.0, "fallback (B200_PROFILING.md)")
    cnt, _ = md.neighbors()
    nb = float(cnt[rk.owned_local].mean())
    by = algo_q6_force_bytes(nb, tb) * nloc
    ach = by / (stage_ms[5] * 1e-3) / 1e9
    roof = {"kernel": "k_q6_force_g (stage apply_forces of this rank: held atoms = owned + halo)", "bound": "hbm", "achieved": ach,
            "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": None, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": by, "kernel_ms": float(stage_ms[5]), "mean_neighbours": nb}
    cfg_ = describe(w, precision)
    cfg_["parallelism"] = (f"slab decomposition along c over {dworld} rank(s): rank {drank} owns {int(rk.owned_local.sum())} atoms and holds "
                           f"{nloc} (halo 2 (rc + skin) = {rk.reach:.2f} A on either side, global coordinates, global box); one all-reduce "
                           f"of {w.ncv} double(s) per step" + ("; THIS LINE: that rank's share alone on one GPU, no all-reduce (--as-rank)" if solo else ""))
    cfg_["hills"] = f"{w.n_hills} seeded hills (no well-tempered replay in this mode)"
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f32" if precision == 32 else "f64", "data": "synthetic", "config": cfg_, "clocks": clocks,
            "gpu_launches": int(launches),
            "e2e": {"value": natoms_job * ke / (e2e_ms_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(pos_h.nbytes + F_h.nbytes),
                    "d2h_bytes_per_step": int(F_h.nbytes + 8 * w.ncv), "ms_per_step": e2e_ms_max / ke},
            "roofline": roof, "stages_ms": {n: float(v) for n, v in zip(names, stage_ms)},
            "decomposition": {"world": dworld, "rank": drank, "owned": int(rk.owned_local.sum()), "held": int(nloc),
                              "fill_fraction": domain.fill_fraction(w.box, rk.reach, dworld), "solo": bool(solo)},
            "state": {"cv": [float(x) for x in cv_h], "sticky": status}}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_peaks(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --peaks needs a CUDA device")
    sampler = ClockSampler(0)
    sampler.start()
    pk = measure_peaks()
    for _ in range(3):                        # keep the SMs busy long enough for a few clock samples
        measure_peaks()
    print(json.dumps({"peaks": pk, "clocks": sampler.stop(), "gpu": torch.cuda.get_device_name(0)}), flush=True)


def main():
    args = parse()
    if args.peaks:
        run_peaks(args)
        return
    if args.impl == "reference":
        run_reference(args)
    elif args.decompose:
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
