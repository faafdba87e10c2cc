#!/usr/bin/env python
"""bench.py -- particle-steps/s of the TILD particle-mesh step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One "step" = one pass of the whole hot path (sort cadence, spread, R2C, fused k-space, C2R, interpolation +
bonds + GJF) over the workload's particles.  Default workload: C4 (8,388,608 particles, 256^3 grid, P=4),
the configuration the BASELINE metric's roofline target is quoted on; it fits one GPU.  Multi-GPU is
"replicas only": every rank runs an independent replica, no data-path collective.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the
same workload; it is a deliberately slow baseline, not the target.
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
sys.path.insert(0, ROOT)

from paper_2302_02474_b200 import inputs  # noqa: E402

METRIC = "particle_steps_per_sec"
UNIT = "particle-steps/s"


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def algorithmic_bytes(cfg):
    """SURVEY 8(d) / DESIGN.md: bytes the method must move per step, per stage."""
    n, S, M = cfg.n, cfg.n_species, cfg.M
    Mk = cfg.grid[0] * cfg.grid[1] * (cfg.grid[2] // 2 + 1)
    return {"spread": 16 * n + 4 * S * M, "kspace": 32 * S * Mk, "interp": 12 * S * M + 52 * n}


def sample_config(cfg):
    """The same recipe at 1/64 of the volume and particle count (same density, same h, same P): used for the ONE-CORE
    oracle figure of the big workloads, where a full-size single-core step would take about a minute."""
    if cfg.n <= 70000:
        return cfg, "the full workload"
    scale = 1.0 / 64.0
    box = cfg.box[0] / 4.0
    grid = cfg.grid[0] // 4
    s = inputs.scaled(cfg, scale, box, grid, name=cfg.name + "_sample64")
    return s, (f"same recipe at 1/64 volume: {s.n} particles, box {box:g}^3, grid {grid}^3, P={cfg.order} "
               f"(same density and mesh spacing)")


class OracleRun:
    """The CPU oracle (oracle/, as it stands) on one workload: state kept between calls so that steps can be timed
    one batch at a time."""

    def __init__(self, cfg, threads=None):
        from oracle import tild_oracle as orc
        self.orc, self.cfg = orc, cfg
        if threads:
            orc.set_threads(threads)
        self.cores = orc.get_threads()
        st = inputs.make_state(cfg)
        self.st = st
        self.p = orc.OracleParams(cfg.n, cfg.n_species, cfg.box, cfg.grid, cfg.order, np.array(cfg.chi), cfg.kappa, cfg.sigma2,
                                  k_bond=cfg.k_bond, r0_bond=cfg.r0_bond, dt=cfg.dt, gamma=cfg.gamma, kT=cfg.kT, mass=cfg.mass,
                                  seed=cfg.philox_seed)
        self.x, self.v = st.x.astype(np.float64), st.v.astype(np.float64)
        self.f = orc.force(self.p, self.x, st.type, st.bond_partner)
        self.step = 0

    def run(self, nsteps):
        """Advances nsteps; returns seconds."""
        t0 = time.perf_counter()
        self.x, self.v, self.f = self.orc.run(self.p, self.x, self.v, self.st.type, self.st.bond_partner, self.step, nsteps, f=self.f)
        self.step += nsteps
        return time.perf_counter() - t0


def oracle_rate(cfg, budget_s, max_steps, threads=None):
    """particle-steps/s of the oracle on cfg: one step to size the run, then as many more as fit in budget_s (at most
    max_steps in all).  Returns (rate, ms per step, cores, steps timed)."""
    o = OracleRun(cfg, threads)
    t1 = o.run(1)
    more = int(max(0, min(max_steps - 1, (budget_s - t1) // max(t1, 1e-6))))
    t = t1 + (o.run(more) if more > 0 else 0.0)
    k = 1 + more
    return cfg.n * k / t, 1e3 * t / k, o.cores, k


def cpu_baseline(cfg):
    """The oracle timed on the box's host cores: FULL-SIZE workload on all cores (>= 3 steps for the big configs) and a
    one-core figure (full size when a step takes under ~10 s on one core, else the 1/64-volume sample)."""
    rate, ms, cores, k = oracle_rate(cfg, budget_s=18.0, max_steps=50 if cfg.n < 2e6 else 3)
    scfg, what = sample_config(cfg)
    r1, ms1, _, k1 = oracle_rate(scfg, budget_s=8.0, max_steps=20, threads=1)
    from oracle import tild_oracle as orc
    orc.set_threads(cores)
    return {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "ms_per_step": ms,
            "sample": f"the full workload ({cfg.n} particles, grid {cfg.grid[0]}^3), {k} steps on {cores} cores",
            "one_core": {"value": r1, "unit": UNIT, "cores": 1, "ms_per_step": ms1, "sample": f"{what}; {k1} steps"}}


def replica_seeds(cfg, rank):
    """Independent replica per rank: same recipe, rank-specific input and Philox seeds."""
    return cfg.input_seed + 7919 * rank, cfg.philox_seed + rank


def max_over_ranks(dist, value, device):
    """Device time of the slowest replica; `dist` is torch.distributed or None (single process)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(n, steps, world, ms_total):
    """Whole-job particle-steps/s: every rank advanced n particles by `steps` steps in ms_total (max over ranks)."""
    return world * n * steps / (ms_total * 1e-3)


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def reference_arm(args, cfg):
    """--impl reference: the oracle on the FULL-SIZE workload, all host cores.  A C4 step takes ~5 s, so the run is
    bounded: W' = min(W, 1) warm-up steps and K' = as many of the K steps as fit in ~100 s; the rate is per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    o = OracleRun(cfg)
    if args.warmup > 0:
        o.run(1)
    t1 = o.run(1)
    more = int(max(0, min(max(1, args.steps) - 1, (100.0 - t1) // max(t1, 1e-6))))
    t = t1 + (o.run(more) if more > 0 else 0.0)
    k = 1 + more
    value, ms = cfg.n * k / t, 1e3 * t / k
    what = f"the full workload ({cfg.n} particles, grid {cfg.grid[0]}^3); {k} of the {args.steps} steps timed on {o.cores} cores"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "n": cfg.n, "grid": list(cfg.grid), "order": cfg.order, "species": cfg.n_species,
                   "steps_timed": k},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": o.cores, "kind": "oracle", "sample": what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def ours_arm(args, cfg):
    import torch
    from paper_2302_02474_b200 import tild

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # independent replica per rank: same recipe, rank-specific seeds
    in_seed, ph_seed = replica_seeds(cfg, rank)
    st = inputs.make_state(cfg, seed=in_seed)
    # --extras: the SURVEY 8(f) rows that ride on extra meshes (per-particle charges: 1 mesh; Maier-Saupe: 5 tensor meshes)
    xkw, xflags = {}, 0
    if args.extras != "none":
        xflags = tild.FLAG_EXTRAS
        if args.extras in ("charges", "both"):
            xkw.update(bjerrum=1.0, a_charge=0.5)
        if args.extras in ("ms", "both"):
            xkw.update(mu_ms=2.5)
    xd, vd = torch.from_numpy(st.x).cuda(), torch.from_numpy(st.v).cuda()
    td, bd = torch.from_numpy(st.type).cuda(), torch.from_numpy(st.bond_partner).cuda()

    def make_engine(flags, stream=None):
        e = tild.Tild(tild.params_from_config(cfg, flags=flags | args.flags | xflags, seed=ph_seed, resort_every=args.resort_every,
                                              tile_shape=args.tile_shape, **xkw), device=f"cuda:{local}", stream=stream)
        if args.extras in ("charges", "both"):      # zero-mean random charges, a third of the particles neutral
            q = np.random.default_rng(in_seed + 5).normal(size=cfg.n).astype(np.float32)
            q[::3] = 0.0
            q -= q.mean()
            e.tild_set_charges(torch.from_numpy(q).cuda())
        if args.extras in ("ms", "both"):           # every second bead with a next bead is an LC centre oriented along that bond
            msp = -np.ones(cfg.n, dtype=np.int32)
            centres = np.where(st.bond_partner[:, 1] >= 0)[0][::2]
            msp[centres] = st.bond_partner[centres, 1]
            e.tild_set_ms_partners(torch.from_numpy(msp).cuda())
        return e

    # Pass 1, the headline: the library as a user gets it (no stage timers: tild_step replays its steps as CUDA graphs), on
    # a stream of its own (the legacy default stream cannot be captured).  W warm-up steps, then exactly K timed steps.
    side = torch.cuda.Stream(device=f"cuda:{local}")
    with torch.cuda.stream(side):
        eng = make_engine(0, stream=side)
        eng.tild_set_state(xd, vd, td, bd, 0)
        eng.tild_step(args.warmup)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    l0 = eng.tild_launch_count()
    with torch.cuda.stream(side):
        e0.record(side)
        eng.tild_step(args.steps)
        e1.record(side)
    barrier()
    launches = eng.tild_launch_count() - l0
    clocks = sampler.stop()
    eng.close()
    # Pass 2, the per-stage times: the same W + K steps with TILD_FLAG_TIMING (eager launches, CUDA events around every stage)
    eng = make_engine(tild.FLAG_TIMING)
    eng.tild_set_state(xd, vd, td, bd, 0)
    eng.tild_step(args.warmup)
    eng.tild_get_timings()                         # synchronises and clears the stage timers
    barrier()
    eng.tild_step(args.steps)
    barrier()
    ms_total = max_over_ranks(dist, e0.elapsed_time(e1), "cuda")
    stage_ms, nst = eng.tild_get_timings()
    value = aggregate_value(cfg.n, args.steps, world, ms_total)

    # end to end through the C-ABI with HOST buffers: every step copies the batch in and the result out.  Two figures: the
    # pipelined calls (tild_run_host_submit / _wait: the copies of consecutive, independent batches overlap the kernels) and
    # the synchronous tild_run_host (one batch at a time, nothing overlaps)
    e2e = None
    if not args.no_e2e:
        xh, vh = torch.from_numpy(st.x.copy()).pin_memory(), torch.from_numpy(st.v.copy()).pin_memory()
        th, bh = torch.from_numpy(st.type.copy()).pin_memory(), torch.from_numpy(st.bond_partner.copy()).pin_memory()
        xo = [torch.empty_like(xh).pin_memory() for _ in range(3)]
        vo = [torch.empty_like(vh).pin_memory() for _ in range(3)]
        reps = max(1, min(args.steps, args.e2e_steps))
        # a context on a stream of its own (the copy streams must not synchronise with the legacy default stream), no stage timers
        eng_t, eng = eng, tild.Tild(tild.params_from_config(cfg, flags=tild.FLAG_HOST_PIPELINE | args.flags, seed=ph_seed,
                                                           resort_every=args.resort_every, tile_shape=args.tile_shape),
                                    device=f"cuda:{local}", stream=side)
        eng.tild_run_host_submit(xh, vh, th, bh, 0, 1, xo[0], vo[0])    # warm-up
        eng.tild_run_host_wait()
        barrier()
        t0 = time.perf_counter()
        for r in range(reps):
            eng.tild_run_host_submit(xh, vh, th, bh, r, 1, xo[r % 3], vo[r % 3])   # H2D + set_state + 1 step + read-out + D2H
            if r >= 2:
                eng.tild_run_host_wait()                 # results of batch r - 2 are in host memory
        for _ in range(min(reps, 2)):
            eng.tild_run_host_wait()
        barrier()
        dt = max_over_ranks(dist, time.perf_counter() - t0, "cuda")
        xs_, vs_ = xh.clone().pin_memory(), vh.clone().pin_memory()
        sreps = max(1, min(reps, 3))
        eng.tild_run_host(xs_, vs_, th, bh, 0, 1)    # warm-up
        barrier()
        t0 = time.perf_counter()
        for r in range(sreps):
            eng.tild_run_host(xs_, vs_, th, bh, r, 1)
        barrier()
        dts = max_over_ranks(dist, time.perf_counter() - t0, "cuda")
        eng.close()
        eng = eng_t
        e2e = {"value": world * cfg.n * reps / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(xh.nbytes + vh.nbytes + th.nbytes + bh.nbytes),
               "d2h_bytes_per_step": int(xh.nbytes + vh.nbytes), "steps": reps,
               "synchronous": {"value": world * cfg.n * sreps / dts, "steps": sreps,
                               "note": "tild_run_host(nsteps=1): one batch at a time, copies and kernels one after the other"},
               "note": "tild_run_host_submit(nsteps=1) + tild_run_host_wait per step, up to three batches in flight: H2D of (x,v,type,bonds), "
                       "sort, one step, F(x) for v, v/x read back; copies of consecutive batches overlap the kernels"}

    if rank != 0:
        return
    peak, peak_src = measured_peak_gbs()
    alg = algorithmic_bytes(cfg)
    stages = {}
    for k in ("spread", "kspace", "interp"):
        gbs = alg[k] / (stage_ms[k] * 1e-3) / 1e9 if stage_ms[k] > 0 else 0.0
        stages[k] = {"ms": stage_ms[k], "alg_bytes": alg[k], "gbs": gbs, "frac": gbs / peak,
                     "traffic": ncu_traffic(cfg.name, k)}
    if not (args.flags & tild.FLAG_PLAIN_FFT) and cfg.n_species <= 4 and cfg.grid[0] in (16, 32, 64, 128, 256):
        stages["kspace"]["note"] = ("fused x-transform kernel: this stage also does the x passes of all 4S FFTs; "
                                    "fft_fwd / fft_inv are the (y, z) passes only")
    dom = max(stages, key=lambda k: stages[k]["ms"])
    three_ms = sum(stages[k]["ms"] for k in stages)
    three_gbs = sum(alg.values()) / (three_ms * 1e-3) / 1e9 if three_ms > 0 else 0.0
    roofline = {"bound": "hbm", "kernel": dom, "achieved": stages[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": stages[dom]["gbs"] / peak, "traffic": ncu_traffic(cfg.name, dom),
                "traffic_source": {k: TRAFFIC.get(k) for k in ("commit", "date", "command")} if TRAFFIC else None,
                "peak_source": peak_src,
                "stages": stages,
                "spread_kspace_interp": {"ms": three_ms, "gbs": three_gbs, "frac": three_gbs / peak,
                                         "frac_of_8TBs_nominal": three_gbs / 8000.0}}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(cfg)
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "n": cfg.n, "grid": list(cfg.grid), "order": cfg.order, "species": cfg.n_species,
                   "resort_every": args.resort_every, "extras": args.extras, "l2": "inputs larger than L2 (no flush needed)"
                   if sum(alg.values()) > 2 * 126e6 else "working set fits L2; steady-state numbers",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "mode": "value / ms_per_step: tild_step as a user calls it (CUDA-graph replay, no stage timers) on a stream of its own; "
                "stage_ms / roofline: a second pass of the same W + K steps with TILD_FLAG_TIMING (eager launches, events per stage)",
        "stage_ms": stage_ms, "stage_steps_timed": nst,
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
    }))
    if dist is not None:
        dist.destroy_process_group()


def load_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the `ncu --set full` capture recorded in
    profiles/traffic_c4.json (commit, date and command are in the file and echoed into the bench line, so a figure
    that is older than the kernels is visible).  {} when the file is missing."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic_c4.json")) as f:
            return json.load(f)
    except Exception:
        return {}


TRAFFIC = load_traffic()


def ncu_traffic(workload, stage):
    if TRAFFIC.get("workload") != workload:
        return None
    ks = TRAFFIC.get("stages", {}).get(stage)
    if not ks:
        return None
    return float(sum(k["dram_bytes_read"] + k["dram_bytes_write"] for k in ks))


def windows_arm(args, cfg):
    """Per-stage times over successive windows of 20 steps of one run (how the step time evolves with the length of the
    run: the memory order of chain neighbours between re-sorts, profiles/r2_variants.md).  One JSON line per window."""
    import torch
    from paper_2302_02474_b200 import tild
    st = inputs.make_state(cfg)
    eng = tild.Tild(tild.params_from_config(cfg, flags=tild.FLAG_TIMING | args.flags, resort_every=args.resort_every))
    d = lambda a: torch.from_numpy(a).cuda()
    eng.tild_set_state(d(st.x), d(st.v), d(st.type), d(st.bond_partner), 0)
    eng.tild_step(max(args.warmup, 0))
    eng.tild_get_timings()
    for w in range(args.windows):
        eng.tild_step(20)
        ms, nst = eng.tild_get_timings()
        print(json.dumps({"window": w, "steps": nst, "workload": cfg.name, "flags": args.flags,
                          "stage_ms": {k: round(v, 4) for k, v in ms.items()}}), flush=True)


def sweep_arm(args):
    """C5 roofline sweep (BASELINE.json configs[4]): grid x order x memory order, 50 steps per point, per-stage times.
    Prints one JSON line per point; not the headline bench line."""
    import torch
    from paper_2302_02474_b200 import tild
    peak, _ = measured_peak_gbs()
    for grid in (128, 192, 256):
        for order in (1, 2, 3, 4):
            for mo in ("random", "sorted"):
                cfg = inputs.c5(grid=grid, order=order, memory_order=mo)
                st = inputs.make_state(cfg)
                eng = tild.Tild(tild.params_from_config(cfg, flags=tild.FLAG_TIMING))
                d = lambda a: torch.from_numpy(a).cuda()
                eng.tild_set_state(d(st.x), d(st.v), d(st.type), d(st.bond_partner), 0)
                eng.tild_step(10)
                eng.tild_get_timings()
                eng.tild_step(cfg.steps)
                ms, nst = eng.tild_get_timings()
                alg = algorithmic_bytes(cfg)
                three = sum(ms[k] for k in alg)
                print(json.dumps({"sweep": "C5", "grid": grid, "order": order, "memory_order": mo, "steps": nst,
                                  "stage_ms": {k: round(v, 4) for k, v in ms.items()},
                                  "particle_steps_per_sec": cfg.n / (ms["total"] * 1e-3),
                                  "frac": {k: alg[k] / (ms[k] * 1e-3) / 1e9 / peak for k in alg},
                                  "spread_kspace_interp_frac": sum(alg.values()) / (three * 1e-3) / 1e9 / peak}), flush=True)
                eng.close()
                del eng


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--resort-every", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--flags", type=int, default=0, help="extra TILD_FLAG_* bits (kernel A/B runs)")
    ap.add_argument("--tile-shape", type=int, default=0, help="tild_params.tile_shape = TY | TZ << 8 (0 = default 8x16x32)")
    ap.add_argument("--extras", default="none", choices=["none", "charges", "ms", "both"],
                    help="per-particle charges and / or Maier-Saupe on their extra meshes (not the headline workload)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--windows", type=int, default=0, help="print per-stage times for this many successive windows of 20 steps")
    ap.add_argument("--sweep", action="store_true", help="run the C5 roofline sweep instead of the headline bench")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    cfg = inputs.CONFIGS[args.workload]
    if args.sweep:
        return sweep_arm(args)
    if args.windows > 0:
        return windows_arm(args, cfg)
    if args.impl == "reference":
        reference_arm(args, cfg)
    else:
        ours_arm(args, cfg)


if __name__ == "__main__":
    main()
