#!/usr/bin/env python
"""bench.py -- ns/particle/timestep of the particle hot path (push + deposit) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--shrink 1] [--impl ours|reference]

One "step" = one pass of the whole hot path over the synthetic plasma: zero J, ent_step for every species (serial host
loop over species), periodic ghost fold, plus ent_sort every --sort-every steps (inside the timed region).
The top-level numbers are the workload of --workload (default C3, the configuration BASELINE.json's metric is quoted on);
without --workload the same line carries `per_config`: C4 sorted, C4 shuffled (its first ent_sort timed alone), C5, C2, C1.
N > 1: one process per GPU (torchrun), every rank pushes an independent replica of the workload ("replicas only",
DESIGN.md): no data-path collective, weak scaling, time = max over ranks.
Prints ONE JSON line (rank 0).  --impl reference times the fp64 CPU oracle on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ns_per_particle_per_timestep_push_plus_deposit"
UNIT = "ns/particle/step"
# algorithmic bytes: read the full record + write the changed fields, fused and in place
PARTICLE_BYTES = {("cart", 3): 60, ("cart", 2): 52, ("axisym", 2): 60}
GRID_BYTES_PER_CELL = 24 + 24            # E,B read once; J read-modify-write (3 comps x (4 + 4) B)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"




def _committed_traffic(workload, mode):
    """(DRAM bytes, warp instructions) per launch of the dominant kernel and their source from the committed ncu capture table
    (profiles/r2_traffic.csv), or (None, None, None)"""
    import csv
    p = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    try:
        for row in csv.DictReader(open(p)):
            if row["workload"] == workload and row["mode"] == mode:
                wi = row.get("warp_instructions_per_launch")
                return float(row["dram_bytes_per_launch"]), (float(wi) if wi else None), row["source"]
    except OSError:
        pass
    return None, None, None


def _issue_ceiling(warp_instr, k_ms, sm_max_mhz, alg_bytes, peak_gbs):
    """Second ceiling of the step kernel (DESIGN.md sect. 5): a B200 issues at most 148 SMs x 4 schedulers x 1 warp instruction per
    cycle.  With the warp instructions of one launch (committed ncu capture) this gives the issue rate the launch reached and the
    fraction of the HBM roofline the same instruction stream could reach at 100 % issue."""
    if not warp_instr or not sm_max_mhz:
        return None
    peak = 148 * 4 * sm_max_mhz * 1e6                       # warp instructions per second
    rate = warp_instr / (k_ms * 1e-3)
    t_min = warp_instr / peak                               # seconds per launch at 100 % issue
    return {"warp_instructions_per_launch": warp_instr, "achieved_ginst_s": rate / 1e9, "peak_ginst_s": peak / 1e9, "frac": rate / peak,
            "hbm_frac_at_full_issue": alg_bytes / t_min / 1e9 / peak_gbs,
            "note": "148 SMs x 4 schedulers x SM clock; instruction count from the committed ncu capture named in traffic_source"}


def max_over_ranks(value: float, device) -> float:
    """time-like quantities are reduced with MAX over the ranks of the job (no-op for a single process)"""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def _load_workload(name, shrink, device, rank=0):
    from paper_2511_17710_b200 import synth
    if name == "C4s":
        return synth.config4(shrink, device=device, shuffled=True)
    return synth.CONFIGS[name](shrink, device=device)


class ClockSampler:
    """nvidia-smi sampled every 10 ms during the timed region (B200_PROFILING.md clocks line); short workloads repeat their timed
    region until it lasts >= 0.5 s so that the sampler sees it"""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "10"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def _oracle_sample(name, target_particles=20_000_000):
    """a bounded sample of the same recipe for the CPU oracle: the workload with every grid extent divided by `shrink`"""
    full = {"C1": 65536, "C2": 2097152, "C3": 134217728, "C4": 536870912, "C4s": 536870912, "C5": 268435456}[name]
    D = 3 if name in ("C3", "C4", "C4s") else 2
    shrink = 1
    while full / (shrink ** D) > target_particles:
        shrink *= 2
    return shrink


def _cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def time_oracle(name, steps, warmup, single_thread_too=False, target_particles=20_000_000):
    """fp64 CPU oracle (oracle/orc.c, as it stands) on a bounded sample; returns a dict"""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import parity as P
    from oracle import orc
    shrink = _oracle_sample(name, target_particles)
    wl = _load_workload(name, shrink, "cpu")
    og = P.grid_to_orc(orc, wl.grid)
    F = P.fields_to_orc(wl.fields)
    parts = [P.species_to_orc(orc, sp) for sp in wl.species]
    J = orc.zeros_current(og)
    npart = sum(p.n for p in parts)

    def one(ps):
        for j in J:
            j[...] = 0.0
        for sp, p in zip(wl.species, ps):
            orc.step(og, F, p, J, sp.q, sp.m, wl.dt)
        orc.fold_current(og, J)
    for _ in range(warmup):
        one(parts)
    t0 = time.perf_counter()
    for _ in range(steps):
        one(parts)
    dt = time.perf_counter() - t0
    out = {"value": dt / (npart * steps) * 1e9, "cores": orc.num_threads(), "ms_per_step": dt / steps * 1e3, "cpu_model": _cpu_model(),
           "host_cores_available": len(os.sched_getaffinity(0)),
           "sample": f"{name} recipe with every grid extent / {shrink}: grid {tuple(wl.grid.N)}, {npart} particles, {steps} steps",
           "workload": f"{wl.name} ({wl.note})"}
    if single_thread_too:                                     # one thread, 1/64 of the sample's particles, one step
        sub = [orc.Particles(i=[a[::64].copy() for a in p.i], d=[a[::64].copy() for a in p.d], u=[a[::64].copy() for a in p.u],
                             w=p.w[::64].copy(), phi=None if p.phi is None else p.phi[::64].copy(), tag=None if p.tag is None else p.tag[::64].copy())
               for p in parts]
        prev = orc.set_num_threads(1)
        t0 = time.perf_counter()
        one(sub)
        out["single_thread_value"] = (time.perf_counter() - t0) / sum(p.n for p in sub) * 1e9
        out["single_thread_sample"] = "every 64th particle of the sample, one step, 1 thread"
        orc.set_num_threads(prev)
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # exactly K timed steps after W warm-up steps, each on a bounded sample of the workload: ~0.75 s per step at 1.7e7 particles on
    # 16 cores; the sample shrinks for large K so that the whole run stays within a few minutes
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    target = 20_000_000 if steps + warmup <= 40 else int(20_000_000 * 40 / (steps + warmup))
    r = time_oracle(args.workload or "C3", steps, warmup, target_particles=target)
    v = r["value"]
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps, "warmup": warmup,
            "ms_per_step": r["ms_per_step"], "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": r["workload"], "note": "fp64 CPU oracle (oracle/orc.c, as it stands) on a bounded sample of the workload"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"], "cpu_model": r["cpu_model"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def measure(args, name, env, want_e2e):
    """times one workload on this rank's GPU; returns the dict of its numbers"""
    import torch
    import torch.distributed as dist
    from paper_2511_17710_b200 import binding as bind, synth
    rank, world, local, dev, peak, peak_src = env
    wl = _load_workload(name, args.shrink, dev, rank)
    g = wl.grid
    eg = bind.Grid(D=g.D, N=tuple(g.N), bc=tuple(g.bc), kind=g.kind, xmin=tuple(g.xmin), xmax=tuple(g.xmax), r0=g.r0,
                   vartheta=g.vartheta)
    stream = torch.cuda.current_stream()
    ctx = bind.ent_create(local, stream)
    bind.ent_set_option(ctx, bind.OPT_STEP_IMPL, args.step_impl)
    bind.ent_set_option(ctx, bind.OPT_SORT_MODE, args.sort_mode)
    if args.tile:
        for k, t in zip((bind.OPT_TILE_1, bind.OPT_TILE_2, bind.OPT_TILE_3), (int(x) for x in args.tile.split(","))):
            bind.ent_set_option(ctx, k, t)
    bind.ent_set_grid(ctx, eg)
    absorb = any(b == synth.ABSORB for b in g.bc)
    parts, spare = [], []
    for sp in wl.species:
        p = bind.Particles(cell=synth.pack_cell(g, sp.i), d=sp.d, u=sp.u, w=sp.w, phi=sp.phi,
                           tag=torch.ones(sp.n, dtype=torch.uint8, device=dev) if absorb else None, q=sp.q, m=sp.m)
        parts.append(p); spare.append(p.empty_like())
    wl.species = None
    F = wl.fields
    J = bind.zeros_current(eg, dev)
    npart = sum(p.n for p in parts)
    ncell = g.ncells
    pbytes = PARTICLE_BYTES[("cart" if g.kind == synth.CART else "axisym", g.D)]
    fused = args.mode == "sorted"
    paired = args.mode == "pair" and len(parts) == 2 and g.kind == synth.CART
    per_launch = len(parts) if paired else 1             # species advanced by one launch of the dominant kernel
    step_ev, sort_ev = [], []          # (start, end) CUDA events around each ent_step / ent_sort call in the timed region

    def timed(fn, store):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); fn(); b.record(stream); store.append((a, b))

    def do_sort(record):
        for k in range(len(parts)):
            f = lambda: bind.ent_sort(ctx, parts[k], spare[k], None)
            timed(f, sort_ev) if record else f()
            parts[k], spare[k] = spare[k], parts[k]

    def one_step(it, record):
        if not fused and args.sort_every > 0 and it > 0 and it % args.sort_every == 0:
            do_sort(record)
        bind.ent_zero_current(ctx, J)
        if paired:                                           # both species of the pair plasma through one launch of the tiled kernel
            f = lambda: bind.ent_step_pair(ctx, F, parts[0], parts[1], J, wl.dt)
            timed(f, step_ev) if record else f()
        for k in range(0 if paired else len(parts)):
            if fused:                                    # fused step + re-bin, ping-pong between the two blocks: no ent_sort at all
                def f():
                    bind.ent_step_sorted(ctx, F, parts[k], spare[k], J, wl.dt)
                    parts[k], spare[k] = spare[k], parts[k]
            else:
                f = lambda: bind.ent_step(ctx, F, parts[k], J, wl.dt)
            timed(f, step_ev) if record else f()
        bind.ent_fold_current(ctx, J)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    bind.ent_reserve(ctx, max(p.n for p in parts))
    first_sort, first_direct = [], []
    shuffled = name == "C4s"
    if shuffled:                       # the block arrives in an unrelated order: the direct scatter once (for the record), then the staged form
        timed(lambda: bind.ent_sort(ctx, parts[0], spare[0], None), first_direct)
        bind.ent_set_option(ctx, bind.OPT_SORT_STAGING, 1)
        bind.ent_sort(ctx, parts[0], spare[0], None)          # untimed: allocates the side buffer
        torch.cuda.synchronize()
    for k in range(len(parts)):        # the particles enter the timed region tile-sorted (BASELINE.json configs 3, 4); timed alone
        timed(lambda: bind.ent_sort(ctx, parts[k], spare[k], None), first_sort)
        parts[k], spare[k] = spare[k], parts[k]
    if shuffled:
        bind.ent_set_option(ctx, bind.OPT_SORT_STAGING, 0)
    it = 0
    w0 = time.perf_counter()
    for _ in range(args.warmup):
        one_step(it, False); it += 1
    barrier()
    est = (time.perf_counter() - w0) / max(1, args.warmup)
    reps = max(1, min(2000, int(0.6 / max(est * args.steps, 1e-6)) + 1)) if est * args.steps < 0.5 else 1
    launches0 = bind.ent_get_stat(ctx, bind.STAT_LAUNCHES)
    clocks = ClockSampler(local) if rank == 0 else None
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for r in range(reps):              # the K steps, repeated so that a short workload is sampled by nvidia-smi too
        for _ in range(args.steps):
            one_step(it, r == 0); it += 1
    t1.record(stream)
    barrier()
    ms = t0.elapsed_time(t1) / reps
    launches = (bind.ent_get_stat(ctx, bind.STAT_LAUNCHES) - launches0) // reps
    clk = clocks.stop() if clocks else None
    tiled = bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED)
    strays = bind.ent_get_stat(ctx, bind.STAT_STRAYS)
    bad = bind.ent_get_stat(ctx, bind.STAT_BAD_MOVES)
    ms = max_over_ranks(ms, dev)
    ms_per_step = ms / args.steps
    value = ms * 1e6 / (npart * world * args.steps)         # whole job: every rank advances its own replica (weak scaling)

    # ---- roofline of the dominant kernel (the fused gather+push+move+deposit kernel), per launch ----
    k_ms = sum(a.elapsed_time(b) for a, b in step_ev) / max(1, len(step_ev))
    alg_bytes = pbytes * npart / len(parts) * per_launch + GRID_BYTES_PER_CELL * ncell
    achieved = alg_bytes / (k_ms * 1e-3) / 1e9
    mean = lambda ev: (sum(a.elapsed_time(b) for a, b in ev) / len(ev)) if ev else None
    traffic, traffic_src, warp_instr = args.traffic, args.traffic_source, None
    if traffic is None and args.shrink == 1 and not args.tile:
        traffic, warp_instr, traffic_src = _committed_traffic(name, "pair" if paired else ("sorted" if fused else "inplace"))
    out = {"name": name, "value": value, "ms_per_step": ms_per_step, "ms_timed": ms, "reps": reps, "npart": npart, "launches": launches,
           "clocks": clk, "tiled": bool(tiled), "strays": strays, "bad_moves": bad, "kernel_ms": k_ms,
           "sort_ms_per_species": mean(sort_ev), "first_sort_ms_per_species": mean(first_sort), "first_sort_direct_ms": mean(first_direct), "fused": fused, "paired": paired,
           "workload": f"{wl.name} ({wl.note})", "grid": list(g.N), "species": len(parts), "dt": wl.dt, "pbytes": pbytes,
           "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                        "traffic": traffic, "traffic_source": traffic_src,
                        "kernel": ("ent_step_sorted" if fused else "ent_step_pair" if paired else "ent_step") + " (fused gather+push+move+deposit), "
                                  + ("both species of the pair plasma per launch" if paired else "one species per launch"),
                        "kernel_ms": k_ms, "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src,
                        "step_share": k_ms * len(parts) / per_launch / ms_per_step,
                        "issue": _issue_ceiling(warp_instr, k_ms, (clk or {}).get("sm_max_mhz"), alg_bytes, peak)}}

    # ---- step 9: 4 digital filter passes (the count of the paper's magnetosphere runs) + J = conformal J / sqrt(h)
    npass = 4
    bind.ent_filter_current(ctx, J, npass, True)
    fev = []
    for _ in range(5):
        timed(lambda: bind.ent_filter_current(ctx, J, npass, True), fev)
    torch.cuda.synchronize()
    f_ms = mean(fev)
    f_bytes = 24.0 * ncell * npass                           # every pass reads and writes the three components once
    out["current_filter"] = {"passes": npass, "ms": f_ms, "algorithmic_bytes": f_bytes, "achieved_gbs": f_bytes / (f_ms * 1e-3) / 1e9,
                             "frac_of_hbm_peak": f_bytes / (f_ms * 1e-3) / 1e9 / peak, "note": "not part of `value` (sub-steps 3-8 only)"}

    # ---- sub-steps 2/10 and 11: the Yee field solver on a copy of the fields (36 / 48 B per cell)
    Fc = [f.clone() for f in F]
    bind.ent_faraday(ctx, Fc, 0.5 * wl.dt); bind.ent_ampere(ctx, Fc, J, wl.dt, 1e-6)
    fa_ev, am_ev = [], []
    for _ in range(5):
        timed(lambda: bind.ent_faraday(ctx, Fc, 0.5 * wl.dt), fa_ev)
        timed(lambda: bind.ent_ampere(ctx, Fc, J, wl.dt, 1e-6), am_ev)
    torch.cuda.synchronize()
    fa_ms, am_ms = mean(fa_ev), mean(am_ev)
    out["field_solver"] = {"faraday_ms": fa_ms, "ampere_ms": am_ms, "faraday_gbs": 36.0 * ncell / (fa_ms * 1e-3) / 1e9,
                           "ampere_gbs": 48.0 * ncell / (am_ms * 1e-3) / 1e9, "frac_of_hbm_peak": [36.0 * ncell / (fa_ms * 1e-3) / 1e9 / peak,
                           48.0 * ncell / (am_ms * 1e-3) / 1e9 / peak], "note": "not part of `value`; algorithmic bytes 36 / 48 B per cell"}
    del Fc

    # ---- end to end through the host-buffer C-ABI call: H2D of the step's inputs and D2H of its results inside ----
    if want_e2e:
        hp = [p.to("cpu", pin=True) for p in parts]
        hF = [f.cpu().pin_memory() for f in F]
        hJ = [torch.zeros(eg.padded_shape, dtype=torch.float32).pin_memory() for _ in range(3)]
        del parts, spare
        torch.cuda.empty_cache()
        nst = max(1, min(args.steps, args.e2e_steps))
        up = down = 0
        host_pair = len(hp) == 2                                  # both species through the pipelined host call

        def host_step():
            if host_pair:
                return bind.ent_step_host_pair(ctx, hF, hp[0], hp[1], hJ, wl.dt, 1)
            u_ = d_ = 0
            for p in hp:
                a, b = bind.ent_step_host(ctx, hF, p, hJ, wl.dt, 1)
                u_ += a; d_ += b
            return u_, d_
        host_step()                                               # warm-up: staging allocation
        tiled_e2e = bind.ent_get_stat(ctx, bind.STAT_LAST_STEP_TILED)
        barrier()
        w0 = time.perf_counter()
        for _ in range(nst):
            up, down = host_step()
        barrier()
        e_ms = max_over_ranks((time.perf_counter() - w0) * 1e3, dev)
        out["e2e"] = {"value": e_ms * 1e6 / (npart * world * nst), "unit": UNIT, "h2d_bytes_per_step": up, "d2h_bytes_per_step": down,
                      "steps": nst, "ms_per_step": e_ms / nst, "tiled_kernel": bool(tiled_e2e),
                      "call": ("ent_step_host_pair: both species, pinned host buffers -> H2D, ent_sort, ent_step (tiled), D2H, pipelined over three streams"
                               if host_pair else "ent_step_host per species: pinned host buffers -> H2D, ent_sort, ent_step (tiled), D2H")}
        del hp, hF, hJ
    bind.ent_destroy(ctx)
    del F, J, wl
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peak, peak_src = _peaks()
    env = (rank, world, local, dev, peak, peak_src)
    main_wl = args.workload or "C3"
    m = measure(args, main_wl, env, want_e2e=not args.no_e2e)
    npart = m["npart"]
    line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": m["ms_per_step"], "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": m["workload"], "grid": m["grid"], "particles_per_gpu": npart, "species": m["species"],
                       "dt": m["dt"], "shrink": args.shrink, "sorted_at_start": True, "sort_every": 0 if m["fused"] else args.sort_every,
                       "step_call": "ent_step_sorted" if m["fused"] else "ent_step_pair" if m["paired"] else "ent_step", "tiled_kernel": m["tiled"],
                       "timed_region_repeats": m["reps"],
                       "l2": "inputs larger than L2 (no flush needed)" if npart * m["pbytes"] > 4e8 else
                       "inputs smaller than L2: the workload itself is L2-resident (BASELINE.json's size), no flush",
                       "parallelism": "replicas only" if world > 1 else "1 GPU"},
            "clocks": m["clocks"], "gpu_launches": m["launches"], "roofline": m["roofline"],
            "particles_per_second": npart * world * args.steps / (m["ms_timed"] * 1e-3),
            "sort_ms_per_species": m["sort_ms_per_species"], "first_sort_ms_per_species": m["first_sort_ms_per_species"],
            "strays_last_step": m["strays"], "bad_moves": m["bad_moves"]}
    if "e2e" in m:
        line["e2e"] = m["e2e"]
    line["current_filter"] = m["current_filter"]
    line["field_solver"] = m["field_solver"]
    if args.workload is None and not args.no_per_config and world == 1:
        per = []
        for name in ("C4", "C4s", "C5", "C2", "C1"):
            try:
                r = measure(args, name, env, want_e2e=False)
                per.append({"workload": r["workload"], "name": name, "particles": r["npart"], "value": r["value"], "unit": UNIT,
                            "ms_per_step": r["ms_per_step"], "kernel_ms": r["kernel_ms"], "roofline_frac": r["roofline"]["frac"],
                            "achieved_gbs": r["roofline"]["achieved"], "sort_ms_per_species": r["sort_ms_per_species"],
                            "first_sort_ms_per_species": r["first_sort_ms_per_species"], "first_sort_direct_scatter_ms": r["first_sort_direct_ms"],
                            "tiled_kernel": r["tiled"],
                            "timed_region_repeats": r["reps"], "gpu_launches": r["launches"], "clocks": r["clocks"]})
            except Exception as e:                            # e.g. not enough free memory on a smaller part: say so, keep the line
                per.append({"name": name, "error": f"{type(e).__name__}: {e}"})
        line["per_config"] = per
    if rank == 0:
        if not args.no_cpu and world == 1:
            r = time_oracle(main_wl, 2, 1, single_thread_too=True)
            line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
                                    "cpu_model": r["cpu_model"], "host_cores_available": r["host_cores_available"],
                                    "single_thread_value": r["single_thread_value"], "single_thread_sample": r["single_thread_sample"]}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=None, choices=["C1", "C2", "C3", "C4", "C4s", "C5"],
                    help="default: C3 as the headline plus the per_config list of the other configurations")
    ap.add_argument("--shrink", type=int, default=1)
    ap.add_argument("--sort-every", type=int, default=3, help="ent_sort every k steps inside the timed region (0 = never)")
    ap.add_argument("--step-impl", type=int, default=0, help="ENT_OPT_STEP_IMPL: 0 auto, 1 untiled, 2 two-kernel, 3 auto with the one-launch pair step on any grid")
    ap.add_argument("--sort-mode", type=int, default=0, help="ENT_OPT_SORT_MODE: 0 auto (incremental re-bin), 1 always the full sort")
    ap.add_argument("--tile", default="", help="tile extents in cells, e.g. 8,8,4 (ENT_OPT_TILE_*; default: the library's)")
    ap.add_argument("--mode", default="pair", choices=["pair", "sorted", "inplace"],
                    help="pair (default): ent_step_pair (both species per launch where the grid is Cartesian, else as inplace) + ent_sort every "
                         "--sort-every steps; inplace: ent_step per species; sorted: ent_step_sorted (fused step + re-bin, out of place)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel from an ncu --set full capture of THIS build")
    ap.add_argument("--traffic-source", default=None, help="the capture --traffic comes from (file under profiles/, commit)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
