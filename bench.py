#!/usr/bin/env python
"""bench.py — throughput of the tDPD + RBC hot path (all rows of SURVEY.md §8(a)) on B200, one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A "step" is one velocity-Verlet step of the whole system through `tdpd_step`: wrap + cell hash, stable radix sort,
cell table + reorder, non-bonded pair kernel, membrane kernel (second stream), fused integrator.
Default workload: BASELINE.json config 5 (128^3 box, 6.29 M solvent particles + 1000 RBCs, two species), the
configuration BASELINE.json names "for peak throughput and ncu roofline capture"; its state (>300 MB) is larger than
the 126 MB L2, so no flush is needed between steps.  Smaller configs (--config 1..4) are timed step by step with an
L2 flush (a 256 MB write) between steps.

  value        particle-steps/s, device-timed (CUDA events on the library's pair stream), state resident in HBM
  e2e          the same metric through the C ABI with HOST buffers: every step copies the whole state host->device
               (tdpd_set_state, pinned memory), advances one step and reads it back (tdpd_get_state)
  roofline     the pair kernel (dominant): algorithmic FLOPs of one launch (per-unit budget x the
               exact pair census of the workload) / its CUDA-event duration, against the FP32 peak of DESIGN.md §7
  cpu_baseline the fp64 oracle (oracle/, as it stands) on this box's host cores on a bounded sample of the workload

--impl reference times the oracle alone (there is no reference implementation; the paper ships no code).
Multi-GPU: "replicas only": each rank runs an independent replica, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import tdpd_workloads as W  # noqa: E402  (inputs only)

L2_BYTES = 126 * 1024 * 1024
SM_COUNT, LANES_PER_SM, SM_MAX_MHZ = 148, 128, 1965.0
# FP32 peak of the plain ALUs: 148 SMs x 128 lanes x 2 FLOP (FMA) x 1.965 GHz
FP32_PEAK_TFLOPS = SM_COUNT * LANES_PER_SM * 2 * SM_MAX_MHZ * 1e6 / 1e12
# per-unit algorithmic budget, SURVEY.md §8(d) / DESIGN.md §7: (FLOP with FMA = 2, FP32+INT lane-instructions)
OPS = dict(cand=(8, 7), flux=(8, 7), rflux=(9, 8), force=(28, 21), philox=(0, 70), boxmuller=(10, 18))


# --------------------------------------------------------------------------------------------------------------
def poiseuille_workload(m_s: float = 0.0):
    """SURVEY §8(f) row 4 / PAPER.md:178-184: transient double Poiseuille flow, 256,000 particles in a periodic 40^3 box,
    alpha = 18.75, gamma = 4.5, r_c = r_cc = 1.58, s = 0.41 (general-exponent path of the pair kernel), +-f in the halves."""
    return W.make_fluid("poiseuille", (40.0, 40.0, 40.0), 4.0, seed=W.BASE_SEED + 11, conc="zero", a=18.75, gamma=4.5,
                        s_R=0.41, r_c=1.58, r_cc=1.58, m_s=m_s, body=0.05, body_mode=W.BODY_DOUBLE_POISEUILLE_Z)


def species_workload(ns: int):
    """SURVEY §8(f) row 2 / PAPER.md:218: the pure-fluid benchmark family (density 4, r_c = 1) with N_spec species, on
    config 2's box (32^3, 131,072 particles)."""
    return W.make_fluid(f"fluid32-S{ns}", (32, 32, 32), 4.0, seed=W.BASE_SEED + 20 + ns, n_species=ns)


def workload(c: int, rank: int = 0, random_flux: bool = True, kind: str = "config", species: int = 0):
    if kind == "poiseuille":
        w = poiseuille_workload()
    elif species:
        w = species_workload(species)
    else:
        w = W.config(c) if random_flux else W.config(c, m_s=0.0)  # m_s = 0: the paper's own setting
    if rank:  # replicas differ only in the random stream
        w.params = dict(w.params, seed=int(w.params["seed"]) + 7919 * rank)
    return w


def sample_workload(c: int):
    """Bounded sample of config c for the oracle leg: the same recipe, density, parameters and species on a smaller
    box (configs 1-3 are used whole; 4-5 keep the RBC lattice spacing of the full box)."""
    if c in (1, 2, 3):
        return W.config(c), f"config{c}, whole system"
    seed = W.BASE_SEED + c
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    from tdpd_workloads import mesh as _mesh
    if c == 4:
        box, grid = (25.6, 25.6, 32.0), (2, 2, 2)
        ctr = W.lattice_centers(box, grid)
    else:
        box, grid = (25.6, 25.6, 25.6), (2, 2, 2)
        ctr = W.lattice_centers(box, grid, rng, jitter=2.0)
    w = W.make_suspension(f"config{c}-sample", box, 3.0, seed, ctr, _mesh.random_rotations(rng, len(ctr)),
                          n_species=2)
    return w, (f"config{c} recipe on a {box[0]}x{box[1]}x{box[2]} box: {w.n_solvent} solvent + {len(ctr)} RBCs "
               f"(same density, lattice spacing, species and parameters)")


def census(sim, w) -> dict:
    """Exact pair census of the workload at the current positions (directed pairs): candidates of the 27-cell
    stencil from the cell occupancy, pairs within r_c / r_cc from the library's integer census (both parity-tested
    bit-exact against the oracle in tests/test_gpu_parity.py).  Setup only, never timed."""
    b = sim.debug_binning()
    nc = b["ncell"]
    cnt = b["cell_count"].reshape(nc[2], nc[1], nc[0]).astype(np.int64)
    nb = np.zeros_like(cnt)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                nb += np.roll(cnt, (dz, dy, dx), axis=(0, 1, 2))
    cs = sim.debug_neighbor_census()
    return dict(n_cand=int((cnt * nb).sum() - cnt.sum()), n_cc=int(cs["n_rcc"].sum()), n_c=int(cs["n_rc"].sum()),
                cells=[int(x) for x in nc])


def pair_budget(cen: dict, params: dict) -> dict:
    """Algorithmic work of ONE pair-kernel launch."""
    S = int(params["n_species"])
    rf = bool(np.any(np.asarray(params["m_s"])[:S] != 0))
    n_cand, n_cc, n_c = cen["n_cand"], cen["n_cc"], cen["n_c"]
    r_c, r_cc = float(params["r_c"]), float(params["r_cc"])
    n_any = max(n_cc, n_c) if r_cc >= r_c else n_c  # pairs that need at least one Gaussian
    n_rng = n_any if rf else n_c
    n_bm = (n_c if not rf else n_cc * ((S + 1 + 1) // 2)) if r_cc >= r_c else n_c  # Box-Muller calls (2 Gaussians)
    n_philox = n_rng * (2 if (rf and S >= 3) else 1)
    tot = [0, 0]
    for k, cnt in (("cand", n_cand), ("flux", n_cc * S), ("rflux", n_cc * S if rf else 0), ("force", n_c),
                   ("philox", n_philox), ("boxmuller", n_bm)):
        tot[0] += OPS[k][0] * cnt
        tot[1] += OPS[k][1] * cnt
    return dict(flop=tot[0], lane_instr=tot[1])


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for nme, v in zip(names, r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(nme)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                    samples=len(sm), reasons=sorted(reasons))


# --------------------------------------------------------------------------------------------------------------
def run_reference(args) -> dict:
    """The oracle, as it stands, on the host cores (the tier's stand-in for a reference implementation)."""
    import oracle
    oracle.build()
    w, what = sample_workload(args.config)
    o = oracle.Oracle.from_workload(w)
    o.compute_forces(0)
    # bound the run: a step costs about the same as the force evaluation just timed
    t0 = time.perf_counter(); o.step(1); t_step = time.perf_counter() - t0
    budget = 150.0
    steps = max(1, min(args.steps, int(budget / max(t_step, 1e-9))))
    warm = max(0, min(args.warmup, int(0.2 * budget / max(t_step, 1e-9)) - 1))
    if warm:
        o.step(warm)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    v = w.n_total * steps / dt
    cores = oracle.num_threads()
    return {
        "impl": "reference", "metric": "tDPD particle-steps/sec", "value": v, "unit": "particle-steps/s",
        "n_gpus": args.gpus, "steps": steps, "warmup": warm + 1, "ms_per_step": 1e3 * dt / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}", "sample": what, "n_particles": w.n_total},
        "cpu_baseline": {"value": v, "unit": "particle-steps/s", "cores": cores, "kind": "oracle", "sample": what},
        "e2e": {"value": v, "unit": "particle-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def cpu_baseline(c: int, seconds: float = 20.0) -> dict:
    import oracle
    oracle.build()
    w, what = sample_workload(c)
    o = oracle.Oracle.from_workload(w)
    t0 = time.perf_counter(); o.compute_forces(0); t_f = time.perf_counter() - t0
    steps = max(1, min(200, int(seconds / max(t_f, 1e-9))))
    t0 = time.perf_counter(); o.step(steps); dt = time.perf_counter() - t0
    return {"value": w.n_total * steps / dt, "unit": "particle-steps/s", "cores": oracle.num_threads(),
            "kind": "oracle", "sample": f"{what}; {steps} steps, {dt:.1f} s"}


def cpu_baseline_of(w, what: str, seconds: float = 20.0) -> dict:
    import oracle
    oracle.build()
    o = oracle.Oracle.from_workload(w)
    t0 = time.perf_counter(); o.compute_forces(0); t_f = time.perf_counter() - t0
    steps = max(1, min(200, int(seconds / max(t_f, 1e-9))))
    t0 = time.perf_counter(); o.step(steps); dt = time.perf_counter() - t0
    return {"value": w.n_total * steps / dt, "unit": "particle-steps/s", "cores": oracle.num_threads(),
            "kind": "oracle", "sample": f"{what}, whole system; {steps} steps, {dt:.1f} s"}


# --------------------------------------------------------------------------------------------------------------
def aggregate(dist, device, ms, ms_e2e, n):
    """Replicas only: whole-job figures = particles summed over ranks / the slowest rank's device time."""
    import torch
    if dist is None:
        return ms, ms_e2e, float(n)
    t = torch.tensor([ms, ms_e2e], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    m = torch.tensor([float(n)], dtype=torch.float64, device=device)
    dist.all_reduce(m, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(m[0])


def run_ours(args) -> dict | None:
    import torch
    import paper_1611_06163_b200 as T

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    T.load_library()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    c = args.config
    w = workload(c, rank, args.random_flux == "on", args.workload, args.species)
    wname = "poiseuille" if args.workload == "poiseuille" else (f"fluid32-S{args.species}" if args.species else f"config{c}")
    sim = T.Simulation.from_workload(w, device=local, pair_threads=args.pair_threads, list_cap=args.list_cap, pair_split=args.pair_split,
                                    skin=args.skin, nlist_cap=args.nlist_cap, single_stream=args.single_stream)
    n, S = sim.n, sim.ns
    K, Wm = args.steps, max(3, args.warmup)
    state_bytes = n * (16 * 3 + 4 * max(S - 1, 0))
    flush = state_bytes < 2 * L2_BYTES
    stream = sim.stream_pair
    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=f"cuda:{local}") if flush else None

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sim.step(Wm)
    sim.sync()
    cen = census(sim, w)
    bud = pair_budget(cen, w.params)

    def timed_steps():
        """K steps bracketed by CUDA events on the library's pair stream; returns (ms, kernel launches)."""
        barrier()
        l0 = sim.launch_count
        if not flush:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            sim.step(K)
            e1.record(stream)
            sim.sync()
            t = e0.elapsed_time(e1)
        else:
            evs = []
            for _ in range(K):
                with torch.cuda.stream(stream):
                    flush_buf.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                sim.step(1)
                b.record(stream)
                evs.append((a, b))
            sim.sync()
            t = sum(a.elapsed_time(b) for a, b in evs)
        nl = sim.launch_count - l0
        barrier()
        return t, nl

    # ---- device-timed region: K steps as a user runs them (steps replayed as CUDA graphs)
    timed_steps()  # untimed pass with the same call pattern: every CUDA graph the timed pass replays is captured here
    clocks = ClockSampler(local) if rank == 0 else None
    ms, launches = timed_steps()
    # ---- the same K steps again with per-kernel-class CUDA events on the launching streams (plain launches: the
    #      event pairs cannot sit inside a graph): the pair kernel's live duration for the roofline
    sim.set_timing(True)
    ms_timers, _ = timed_steps()
    clk = clocks.stop() if clocks else None
    tim = sim.get_timing()
    sim.set_timing(False)

    # ---- end to end through the C ABI with host buffers (pinned), every step: H2D state, one step, D2H state
    Ke = max(3, min(K, 10))
    pin = lambda wdt: torch.empty((n, wdt), dtype=torch.float32, pin_memory=True).numpy()
    hb = dict(pos=pin(3), vel=pin(3), conc=pin(S))
    sim.get_state(forces=False, out=hb)
    for _ in range(2):
        sim.set_state(hb["pos"], hb["vel"], hb["conc"]); sim.step(1); sim.get_state(forces=False, out=hb)
    barrier()
    t0 = time.perf_counter()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(Ke):
        sim.set_state(hb["pos"], hb["vel"], hb["conc"])
        sim.step(1)
        sim.get_state(forces=False, out=hb)
    b.record(stream)
    sim.sync()
    ms_e2e = max(a.elapsed_time(b), 1e3 * (time.perf_counter() - t0))
    barrier()

    tmax, temax, ntot = aggregate(dist, f"cuda:{local}", ms, ms_e2e, n)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return None

    # ---- roofline of the pair kernel (dominant): measured denominators (tdpd_measure_peaks)
    mp = T.measure_peaks(local)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak, hbm_src = (peaks["hbm_gbs"], "measured") if "hbm_gbs" in peaks else (6650.0, "fallback")
    pair_ms = tim["pair"]["ms"] / max(tim["pair"]["launches"], 1)
    ach = bud["flop"] / (pair_ms * 1e-3) / 1e12
    issue_peak = SM_COUNT * LANES_PER_SM * SM_MAX_MHZ * 1e6  # lane-instructions / s
    kernel_ms = {k: v["ms"] / max(K, 1) for k, v in tim.items()}
    # P4 + X4 + vel (+ Y2 for S > 2) in, F4 (+ Qx) out, per particle
    pair_hbm_bytes = n * (48 + (8 if S > 2 else 0) + 16 + 4 * max(S - 1, 0))
    traffic = None
    try:  # measured DRAM bytes of one launch from the committed ncu capture of the same workload, if there is one
        tj = json.load(open(os.path.join(ROOT, "profiles", "r2_pair_traffic.json")))
        if args.random_flux == "on" and wname in tj and not args.skin:
            traffic = tj[wname]["dram_bytes_per_launch"]
    except Exception:
        pass
    fp32_peak = max(mp["fp32_fma_tflops"], mp["fp32_fma2_tflops"])
    # BASELINE's roofline, all three legs: FLOPs at the FP32 peak, staged bytes at the L2 bandwidth
    # (algorithmic: a 2x2x2-cell brick reads its 4x4x4 halo once, 32 B x 8 per particle), compulsory bytes at HBM
    staged_bytes = n * 32 * 8
    legs = {"flop_ms": bud["flop"] / (fp32_peak * 1e12) * 1e3, "l2_ms": staged_bytes / (mp["l2_read_gbs"] * 1e9) * 1e3,
            "hbm_ms": pair_hbm_bytes / (hbm_peak * 1e9) * 1e3}
    t_roof = max(legs.values())
    roof = {
        "kernel": "k_pair", "bound": "alu", "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s",
        "frac": t_roof / pair_ms,
        "peak_source": "measured live by tdpd_measure_peaks: FMA microbenchmark, max of scalar fma (%.1f) and packed "
                       "fma.rn.f32x2 / FFMA2 (%.1f TFLOP/s); nominal 148 x 128 x 2 x 1.965 GHz = %.1f"
                       % (mp["fp32_fma_tflops"], mp["fp32_fma2_tflops"], FP32_PEAK_TFLOPS),
        "legs_ms": legs, "l2_read_gbs_measured": mp["l2_read_gbs"], "hbm_read_gbs_measured": mp["hbm_read_gbs"],
        "staged_bytes": staged_bytes,
        "traffic": traffic, "traffic_source": "committed ncu capture (profiles/), not measured in this run",
        "traffic_unit": "bytes per launch (ncu dram read + write)", "algorithmic_bytes": pair_hbm_bytes,
        "ms_per_launch": pair_ms, "flop_per_launch": bud["flop"], "share_of_step": kernel_ms["pair"] / (ms_timers / max(K, 1)),
        "timed": "a second pass of the same K steps with per-kernel CUDA events (plain launches); value comes from the first pass (CUDA graphs)",
        "issue_slot_frac": bud["lane_instr"] / (pair_ms * 1e-3) / issue_peak,
        "hbm_gbs_algorithmic": pair_hbm_bytes / (pair_ms * 1e-3) / 1e9, "hbm_peak_gbs": hbm_peak,
        "hbm_peak_source": hbm_src, "census": cen,
    }
    out = {
        "metric": "tDPD particle-steps/sec", "value": ntot * K / (tmax * 1e-3), "unit": "particle-steps/s",
        "n_gpus": world, "steps": K, "warmup": Wm + K, "ms_per_step": tmax / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": wname, "n_particles": n, "n_rbc": sim.n_rbc, "n_species": S,
                   "box": [float(x) for x in w.params["box"]], "random_flux": bool(np.any(w.params["m_s"][:S] != 0)),
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": ("256 MB flush write between timed steps" if flush else
                          f"no flush: state {state_bytes / 2**20:.0f} MB per side > 126 MB L2")},
        "e2e": {"value": ntot * Ke / (temax * 1e-3), "unit": "particle-steps/s", "steps": Ke,
                "h2d_bytes_per_step": int(n * (6 + S) * 4), "d2h_bytes_per_step": int(n * (6 + S) * 4),
                "what": "per step: tdpd_set_state (pinned host -> device, the whole state), tdpd_step(1), tdpd_get_state "
                        "(device -> pinned host); a state replaced by the host needs F(t) again, so a step costs TWO force "
                        "evaluations by construction (DESIGN.md §7)"},
        "gpu_launches": int(launches), "clocks": clk, "roofline": roof,
        "kernel_ms_per_step": kernel_ms, "ms_per_step_with_timers": ms_timers / K,
        "kernel_ms_note": "CUDA-event time per class per step on its own stream; membrane runs on the second stream concurrently with pair, so its figure includes the time it shares the SMs with the pair kernel",
    }
    if args.skin:
        out["config"]["neighbor_list"] = dict(skin=args.skin, **sim.neighbor_list_stats())
    if not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(c) if wname.startswith("config") else cpu_baseline_of(w, wname)
    if dist is not None:
        dist.destroy_process_group()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--pair-threads", type=int, default=0, help="pair-kernel CTA size override (tuning)")
    ap.add_argument("--pair-split", type=int, default=0, help="pair-kernel threads per particle override (tuning)")
    ap.add_argument("--list-cap", type=int, default=0, help="pair-kernel list capacity override (tuning)")
    ap.add_argument("--workload", default="config", choices=["config", "poiseuille"],
                    help="poiseuille: the paper's transient double-Poiseuille case (256 k particles, s = 0.41)")
    ap.add_argument("--species", type=int, default=0, help="N_spec-species fluid on config 2's box (PAPER.md:218)")
    ap.add_argument("--single-stream", action="store_true",
                    help="membrane kernel on the pair stream instead of its own (shows what the second stream hides)")
    ap.add_argument("--skin", type=float, default=0.0, help="neighbour-list mode: skin radius (0 = bin every step)")
    ap.add_argument("--nlist-cap", type=int, default=0, help="neighbour-list capacity per particle (0 = automatic)")
    ap.add_argument("--random-flux", default="on", choices=["on", "off"],
                    help="off: m_s = 0, the random concentration flux dropped as in the paper (PAPER.md:78)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)), flush=True)
        return
    out = run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
