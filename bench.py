#!/usr/bin/env python
"""bench.py -- MLUPS of the particle-resolved thermal LBM hot path on B200 (one JSON line).

A "step" is one time step of the whole hot path (rows a1-a6 of SURVEY.md 8(a): link build,
bounce-back + momentum exchange, particle update, flag update, fused stream-collide, refill) on
the workload BASELINE.json's metric is quoted on: config 3, 4000 x 4000 fp64 D2Q9+D2Q5 with 4,800
hot particles (seeded synthetic placement, paper_2308_16597_b200/workloads.py).

  value  MLUPS = nx*ny*K / seconds (Eq. 18), state resident in HBM, CUDA events
         around ONE lbm_step(K) call on the library's stream, max over ranks
  e2e    the same metric for a whole job through the public API with HOST buffers: lbm_create ->
         lbm_set_temperature(host T) -> lbm_add_particles(host arrays) -> lbm_step(K) ->
         lbm_get_fields(rho, ux, uy, T to pinned host) + lbm_get_particles, all inside the timed
         region (an LBM state lives on the device between steps, so the host copies of a job are
         its set-up and its read-out; bytes are reported per step = job bytes / K)
  roofline      fused stream-collide kernel: algorithmic bytes / its mean CUDA-event duration
  cpu_baseline  the CPU oracle as it stands, timed on this host on a bounded sample

N > 1 (torchrun): north_star keeps the measured path on one GPU: every rank
runs an independent replica of the workload, no data-path collective; value = all ranks' lattice
updates / max-over-ranks time ("weak").  --slabs cuts ONE lattice into a y-slab per rank instead
(include/lbm.h "y-slabs"; "strong").

--impl reference: times the oracle (single thread, host cores) on a bounded sample of the same
workload; the ratio against it is not a headline (it is a deliberately slow checker).
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "MLUPS (fp64 D2Q9+D2Q5 with particles, 1 B200) and % of HBM roofline"
BYTES_PER_LU = 2 * (9 + 5) * 8     # one read + one write of every population
FLAG_BYTES = 1


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=200)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs[k] (default 3); 5 = the paper's own Table 4 benchmark "
                         "(d = 40, 60 x 80 array; the one workload BASELINE.md has a published number for)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--profile-steps", type=int, default=200)
    ap.add_argument("--slabs", action="store_true",
                    help="cut the lattice into one y-slab per rank (strong scaling: halo rows and the "
                         "force combine cross NVLink every step) instead of independent replicas; "
                         "north_star keeps the headline on one GPU, so this is not the default")
    ap.add_argument("--edge", type=int, default=0,
                    help="config 1 only: particle-free lattice of this edge instead of 1024 "
                         "(same physics and initial-state recipe)")
    return ap.parse_args()


# ---------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi samples DURING the timed region (B200_PROFILING.md, clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        inside = [l for (t, l) in self.lines if t0 <= t <= t1 + 0.1] or [l for _, l in self.lines]
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in inside:
            c = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); power.append(float(c[2]))
            except (ValueError, IndexError):
                continue
            for nme, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm),
                "reasons": sorted(reasons)}


# ---------------------------------------------------------------- oracle (CPU) legs
def oracle_sample_workload(wl, cfg, edge):
    """A bounded sample of config `cfg`: an edge x edge lattice with the same particle number
    density, diameters, density ratio, temperatures, physics and placement recipe."""
    full = wl.config(cfg) if cfg in (0, 1) else None
    if cfg == 0:
        return full
    if cfg == 5:
        c = max(2, edge // 50)
        return wl.paper_table4(cols=c, lines=max(1, (3 * c) // 4), name=f"paper_table4_sample_{50 * c}")
    if cfg == 1:
        import numpy as np
        rng = np.random.default_rng(1)
        j = np.arange(edge, dtype=np.float64)[:, None]
        T = (1.0 - (j + 0.5) / edge) + 1e-3 * rng.uniform(-1.0, 1.0, size=(edge, edge))
        return wl.Workload("config1_sample", edge, edge, full.params, 1, 1, T_init=T)
    spec = {2: (1000, 480, 0.4, 20.0, 20.0), 3: (4000, 4800, 0.3, 20.0, 20.0),
            4: (8192, 20000, 0.0, 12.0, 24.0)}[cfg]
    n_full, np_full, yfrac, dlo, dhi = spec
    npart = max(1, int(round(np_full * (edge / n_full) ** 2)))
    return wl.sedimentation(edge, edge, npart, seed=cfg, y_frac_lo=yfrac, d_lo=dlo, d_hi=dhi,
                            name=f"config{cfg}_sample_{edge}")


def host_gb_free():
    try:
        import psutil
        return psutil.virtual_memory().available / 2 ** 30
    except ImportError:
        return 0.0


# host memory the oracle needs for a full config (three copies of f, g + fields), GB
ORACLE_FULL_GB = {0: 0.1, 1: 1.0, 2: 1.0, 3: 8.0, 4: 32.0, 5: 8.0}


def time_oracle(wl, cfg, edge, steps, warmup):
    """edge = 0: the full config; else a square sample of that edge."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle_binding as ob
    w = wl.config(cfg) if edge == 0 else oracle_sample_workload(wl, cfg, edge)
    o = ob.OracleSim.from_workload(w)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return w, w.nx * w.ny * steps / dt / 1e6, dt


def run_reference(args, wl):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    total = args.steps + args.warmup
    full = wl.config(args.config)
    # the FULL config whenever the oracle can finish it in a few minutes (about 5 MLUPS on one
    # core: 3.3 s per step of config 3) and the host has the memory; else a bounded sample sized
    # so that the whole run ends within ~2 minutes
    full_seconds = full.nx * full.ny * total / 4.5e6
    if full_seconds <= 240.0 and host_gb_free() >= ORACLE_FULL_GB.get(args.config, 8.0) + 4.0:
        edge = 0
    else:
        edge = int(math.sqrt(max(1.0, 120.0 * 1.5e6 / max(total, 1))))
        edge = max(96, min(1000, edge))
    w, val, dt = time_oracle(wl, args.config, edge, args.steps, args.warmup)
    what = "the full config" if edge == 0 else f"{w.nx}x{w.ny} sample of config {args.config}"
    sample = (f"{what} ({w.nx}x{w.ny}, {w.n_particles} particles; samples keep the "
              f"density/diameters/physics/placement recipe), {args.steps} steps after "
              f"{args.warmup} warm-up, single thread")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "MLUPS",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dt / max(args.steps, 1) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name if edge == 0 else f"config{args.config}", "sample": sample,
                       "same_config": edge == 0},
            "cpu_baseline": {"value": val, "unit": "MLUPS", "cores": 1, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": "MLUPS", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------- our arm
def main():
    args = parse_args()
    from paper_2308_16597_b200 import workloads as wl
    if args.impl == "reference":
        run_reference(args, wl)
        return

    import numpy as np
    import torch
    from paper_2308_16597_b200 import binding, replicas
    if args.slabs:
        run_slabs(args, wl)
        return

    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    replicas.init("nccl", dev)

    def barrier():
        replicas.barrier(dev)

    K, W = args.steps, max(args.warmup, 3)
    w = wl.config(args.config)
    if args.edge and args.config == 1:
        w = oracle_sample_workload(wl, 1, args.edge)
        w.name = f"config1_rayleigh_benard_{args.edge}"
    n = w.nx * w.ny
    stream = torch.cuda.current_stream(dev)

    # ---------------- device-resident timing: value
    sim = binding.Simulation.from_workload(w, device=dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    vis = [v for v in os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",") if v.strip()]
    clocks = ClockSampler(vis[local] if local < len(vis) else local)
    clocks.start()
    time.sleep(0.3)                  # nvidia-smi is up and sampling
    # the warm-up runs straight into the timed region: an idle gap here lets the GPU fall back
    # to its idle clocks (120 MHz), and the ramp back up then lands inside the timed steps
    # (measured: one run in four 15-55 us per step slower)
    sim.step(W)
    # one-time plan building outside the timed region (lbm_prepare: band plan, capture, instantiation
    # and upload of the CUDA graphs the timed call replays; no time step is taken)
    sim.prepare(K)
    barrier()
    l0 = sim.kernel_launches()
    t0 = time.perf_counter()
    ev0.record(stream)
    sim.step(K)                      # K time steps, one stream synchronisation at the end
    ev1.record(stream)
    barrier()
    t1 = time.perf_counter()
    launches = sim.kernel_launches() - l0
    ms = ev0.elapsed_time(ev1)
    clk = clocks.stop(t0, t1)
    ms_max = replicas.max_over_ranks(ms, dev)
    value = replicas.whole_job_mlups(n, K, ms_max, world)

    # ---------------- per-kernel CUDA-event durations -> roofline.  Two separate passes after the
    # timed region: (a) strictly sequential on one stream (each kernel alone on the GPU), (b) as
    # benched (particle update chain on its own stream, concurrent with the lattice kernel).
    P = max(min(args.profile_steps, 512), 16)     # (calls of fewer than 16 steps run the plain schedule)

    def profile_pass(overlap):
        sim.set_overlap(overlap)
        sim.step(3)
        sim.profile(True)
        sim.step(P)
        r = sim.profile_results()
        sim.profile(False)
        return {k: (v[0] / v[1] if v[1] else 0.0) for k, v in r.items() if k != "init_collide"}

    seq = profile_pass(False)
    ovl = profile_pass(True)
    band_q = sim.band_rows()     # rows [0, Q) advanced two steps per pass (0: none)
    st = sim.fields()
    flag = st["flag"]
    n_fluid = int((flag == 0).sum())
    # a particle-free lattice advances two steps per launch (k_stream_collide_2step): the launch
    # then carries two lattice updates per node (2 x 224 B algorithmic) while moving ~137 B per
    # update, so its fraction of the 224 B/LU roofline may exceed 1
    # (three per launch with k_stream_collide_3step: 3 x 224 B algorithmic, ~105 B per update moved)
    # (k_stream_collide_3step_tma: the persistent TMA-fed variant, the default from 2^20 nodes)
    three_tma = ovl.get("stream_collide_3step_tma", 0.0) > 0.0 and w.particles is None
    three_step = three_tma or (ovl.get("stream_collide_3step", 0.0) > 0.0 and w.particles is None)
    two_step = three_step or (ovl.get("stream_collide_2step", 0.0) > 0.0 and ovl.get("stream_collide", 0.0) == 0.0)
    kname = ("stream_collide_3step_tma" if three_tma else "stream_collide_3step") if three_step else \
        ("stream_collide_2step" if two_step else "stream_collide")
    per_launch = 3 if three_step else (2 if two_step else 1)
    far_s = seq[kname] * 1e-3
    far_ovl_s = ovl[kname] * 1e-3
    step_ms_seq = sum(seq.values())
    # 14 doubles read + 14 written per fluid node + 1 flag byte per node.
    # With a two-step band the one-step kernel covers the rows from Q up (and row Q-1 in every
    # other step); the band's kernel advances Q*nx nodes by one step per launch on average
    band_rows = band_q if band_q > 0 else (w.ny + band_q if band_q < 0 else 0)   # (< 0: a band under the lid)
    if two_step:
        alg_bytes = per_launch * BYTES_PER_LU * n_fluid
    elif band_rows > 0:
        outside = flag[band_q:] if band_q > 0 else flag[:-band_q]
        # (two steps per pass: the one-step kernel also updates row Q-1 in every other step)
        extra = 0.0 if ovl.get("stream_collide_3step", 0.0) > 0.0 else 0.5
        fluid_top = int((outside == 0).sum()) + extra * w.nx
        alg_bytes = BYTES_PER_LU * fluid_top + FLAG_BYTES * (w.ny - band_rows + extra) * w.nx
    else:
        alg_bytes = BYTES_PER_LU * n_fluid + FLAG_BYTES * n
    band = None
    if band_rows > 0 and not two_step:
        # the band's kernel: three steps per pass (k_stream_collide_3step<BAND>, a third of the tile
        # rows per step) under the suspension by default, else two (k_stream_collide_2step, half)
        bk = "stream_collide_3step" if ovl.get("stream_collide_3step", 0.0) > 0.0 else "stream_collide_2step"
        b_s = ovl[bk] * 1e-3
        band = {"rows": band_rows, "where": "below the suspension" if band_q > 0 else "above the suspension",
                "kernel": "k_" + bk + ("<BAND>" if bk.endswith("3step") else ""), "launches_per_step": 1,
                "steps_per_pass": 3 if bk.endswith("3step") else 2,
                "lattice_updates_per_launch": band_rows * w.nx, "avg_launch_ms": b_s * 1e3,
                "avg_launch_ms_alone": seq[bk],
                "algorithmic_gbs_at_224_B_per_update": BYTES_PER_LU * band_rows * w.nx / b_s / 1e9 if b_s > 0 else None}
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak, peak_src = float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    else:
        peak, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
    # `achieved` is taken in the schedule the timed region runs (the particle chain sharing the
    # GPU with the lattice kernel); the kernel alone on the GPU is reported beside it
    achieved = alg_bytes / far_ovl_s / 1e9 if far_ovl_s > 0 else 0.0
    roofline = {"bound": "hbm", "kernel": "k_" + kname, "lattice_updates_per_launch": per_launch,
                "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": read_traffic() if args.config == 3 else None,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                "avg_launch_ms": far_ovl_s * 1e3, "launches_timed": P,
                "avg_launch_ms_alone": far_s * 1e3,
                "achieved_alone": alg_bytes / far_s / 1e9 if far_s > 0 else 0.0,
                "share_of_sequential_step": seq[kname] / step_ms_seq if step_ms_seq else None,
                "kernel_ms_per_step_sequential": seq, "kernel_ms_per_step_overlapped": ovl,
                "whole_step_frac_of_hbm_roofline": value / world / (peak * 1e9 / BYTES_PER_LU / 1e6),
                # north_star words the roofline as "about 8 TB/s" (nominal): 35,714 MLUPS
                "whole_step_frac_of_nominal_8TBs_roofline": value / world / (8.0e12 / BYTES_PER_LU / 1e6),
                # the same step counted in the method's own bytes (224 B per FLUID node + 1 flag
                # byte per node; solid nodes are never moved) over the step time, against the peak
                "whole_step_frac_fluid_bytes": (BYTES_PER_LU * n_fluid + FLAG_BYTES * n) / (ms_max / K * 1e-3) / 1e9 / peak,
                "two_step_band": band,
                "fluid_fraction": n_fluid / n}
    sim.close()
    del sim
    torch.cuda.empty_cache()

    # ---------------- end to end through the public API with host buffers
    e2e = None
    if not args.no_e2e:
        T_host = torch.empty((w.ny, w.nx), dtype=torch.float64).pin_memory()
        if w.T_init is not None:
            T_host.copy_(torch.from_numpy(np.ascontiguousarray(w.T_init)))
        else:
            T_host.fill_(w.params["T0"])
        outs = {k: torch.empty(n, dtype=torch.float64).pin_memory() for k in ("rho", "ux", "uy", "T")}
        h2d = T_host.numel() * 8
        if w.particles is not None:
            h2d += sum(int(np.asarray(v).nbytes) for v in w.particles.values())
        # one untimed rehearsal of the job (3 steps): every kernel of the set-up and read-out path is
        # loaded, the allocator and the pinned buffers have been used once
        s2 = binding.Simulation(w.nx, w.ny, w.params, device=dev)
        s2.set_temperature(T_host)
        if w.particles is not None:
            s2.add_particles(**w.particles)
        s2.step(3)
        s2.fields(out=outs)
        s2.particles()
        s2.close()
        del s2
        barrier()
        te0 = time.perf_counter()
        s2 = binding.Simulation(w.nx, w.ny, w.params, device=dev)
        tb = [time.perf_counter()]
        s2.set_temperature(T_host)
        tb.append(time.perf_counter())
        if w.particles is not None:
            s2.add_particles(**w.particles)
        tb.append(time.perf_counter())
        s2.step(K)
        tb.append(time.perf_counter())
        res = s2.fields(out=outs)
        pr = s2.particles()
        barrier()
        tb.append(time.perf_counter())
        te = tb[-1] - te0
        stages = dict(zip(("create", "set_temperature", "add_particles", "step", "read_out"),
                          (round(1e3 * (b - a), 3) for a, b in zip([te0] + tb[:-1], tb))))
        d2h = 4 * n * 8 + n + sum(int(v.nbytes) for v in pr.values())
        te_max = replicas.max_over_ranks(te, dev)
        assert np.isfinite(res["rho"]).all()
        e2e = {"value": replicas.whole_job_mlups(n, K, te_max * 1e3, world), "unit": "MLUPS",
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
               "job": "create + set_temperature(host) + add_particles(host) + step(K) + "
                      "get_fields(rho,ux,uy,T,flag -> pinned host) + get_particles",
               "job_seconds": te_max, "job_stages_ms": stages}
        s2.close()

    # ---------------- CPU baseline: the oracle on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # about 15-25 s of single-thread work: the full config where a handful of steps fit
        # (config 3: 5 steps of 3.3 s; configs 0-2: more steps), a sample only for config 4
        if args.config in (0, 1, 2, 3, 5) and host_gb_free() >= ORACLE_FULL_GB[args.config] + 4.0:
            edge = 0
            steps_cpu = {0: 4000, 1: 60, 2: 60, 3: 5, 5: 5}[args.config]
        else:
            edge, steps_cpu = 600, 200
        wc, v, dt = time_oracle(wl, args.config, edge, steps_cpu, 1)
        what = "the full config" if edge == 0 else f"{wc.nx}x{wc.ny} sample of config {args.config}"
        cpu = {"value": v, "unit": "MLUPS", "cores": 1, "kind": "oracle",
               "sample": f"{what} ({wc.nx}x{wc.ny}, {wc.n_particles} particles), {steps_cpu} steps "
                         f"after 1, {dt:.1f} s, single thread of {os.cpu_count()} host cores"}

    # BASELINE.md holds a published number only for the paper's own workload (config 5): 1750 MLUPS
    # on 1x A100 (Table 5) -- another machine's, context rather than target
    vs_baseline = value / 1750.0 if (args.config == 5 and world == 1) else None
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": "MLUPS", "n_gpus": world, "steps": K,
                "warmup": W, "ms_per_step": ms_max / K, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": vs_baseline, "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "nx": w.nx, "ny": w.ny, "particles": w.n_particles,
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": f"inputs larger than L2: {2 * 14 * 8 * n / 1e6:.0f} MB of "
                                 "populations stream through per step (126 MB L2)"
                                 if 2 * 14 * 8 * n > 126e6 * 2 else "working set fits L2: not an HBM-bound configuration",
                           "seed": "numpy default_rng(config index)",
                           "timed_region": "one lbm_step(K) call after lbm_step(W) and lbm_prepare(K) "
                                           "(graphs captured and uploaded beforehand)"},
                "clocks": clk, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "cpu_baseline": cpu,
                "context": {"paper_single_gpu_mlups": 1750, "paper_hardware": "1x A100, OpenACC "
                            "(PAPER.md:271-281; d=40, Pr=5 workload: context, not like-for-like)"}}
        print(json.dumps(line))
    replicas.shutdown()


def run_slabs(args, wl):
    """One y-slab per rank (paper_2308_16597_b200/slabs.py, include/lbm.h "y-slabs"): the same
    metric on a lattice cut along y; per step one all-reduce of 3 doubles per particle and one
    send / recv of `halo` rows x 14 populations with each neighbour."""
    import torch
    from paper_2308_16597_b200 import replicas, slabs
    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    replicas.init("nccl", dev)
    K, W = args.steps, max(args.warmup, 3)
    w = wl.config(args.config)
    sr = slabs.SlabRank(w, rank, world, dev)
    stream = torch.cuda.current_stream(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clocks = ClockSampler(local)
    clocks.start()
    time.sleep(0.3)
    sr.step(W)
    replicas.barrier(dev)
    l0 = sr.sim.kernel_launches()
    t0 = time.perf_counter()
    ev0.record(stream)
    sr.step(K)
    ev1.record(stream)
    replicas.barrier(dev)
    t1 = time.perf_counter()
    launches = sr.sim.kernel_launches() - l0
    ms_max = replicas.max_over_ranks(ev0.elapsed_time(ev1), dev)
    clk = clocks.stop(t0, t1)
    value = w.nx * w.ny * K / (ms_max * 1e-3) / 1e6          # one lattice, all ranks together
    if rank == 0:
        j0, j1 = sr.ranges[0]
        line = {"metric": METRIC, "value": value, "unit": "MLUPS", "n_gpus": world, "steps": K,
                "warmup": W, "ms_per_step": ms_max / K, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "nx": w.nx, "ny": w.ny, "particles": w.n_particles,
                           "parallelism": f"{world} y-slabs of ~{j1 - j0} rows, {sr.halo} ghost rows "
                                          "per face, direct launches (no graphs, no band)",
                           "l2": "inputs larger than L2" if 2 * 14 * 8 * w.nx * w.ny / world > 252e6
                                 else "working set fits L2"},
                "clocks": clk, "e2e": None, "gpu_launches": launches, "roofline": None,
                "cpu_baseline": None}
        print(json.dumps(line))
    sr.close()
    replicas.shutdown()


def read_traffic():
    """dram bytes (read + write) per k_stream_collide launch from the committed ncu --set full
    capture, or None: profiles/traffic.csv, rows `kernel,dram_bytes_per_launch` (see the .md
    beside it for the command)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for row in open(p):
            c = row.strip().split(",")
            if c[0] == "k_stream_collide":
                return float(c[1])
    except (OSError, ValueError, IndexError):
        pass
    return None


if __name__ == "__main__":
    main()
