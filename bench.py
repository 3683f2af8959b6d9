#!/usr/bin/env python
"""Benchmark of the SPH hot path on B200 (driver contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config I] [--pi-kernel P]

A "step" is one symplectic step of the whole hot path (2 neighbour-list builds + 2 particle-interaction
passes + dt reduction + predictor + corrector) on BASELINE.json configs[2]
(3-D dam break, 4 074 144 fluid + 801 128 boundary particles), synthetic and seeded.
Metric: particle interactions per second (the paper's PIPS), whole-job.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "particle_interactions_per_s"
UNIT = "interactions/s"
# Work model fixed in BASELINE.md section 2 / DESIGN.md before measuring:
FLOPS_PER_ACCEPTED = 41.0      # per accepted ordered pair
FLOPS_PER_CANDIDATE = 8.0      # per candidate distance test
CAND_PER_ACCEPTED = {1: 6.45, 2: 3.73, 3: 2.75}   # (2k+1)^3 cells of size 2h/k vs the 2h sphere (k=3: clipped stencil)
CAND_PER_ACCEPTED_2D = {1: 2.865, 2: 1.989, 3: 1.733}   # (2k+1)^2 cells of size 2h/k vs the 2h disc
SM_COUNT, FP32_LANES_PER_SM = 148, 128


def fp32_peak_tflops(sm_mhz: float) -> float:
    """Plain-FMA FP32 peak: 148 SMs x 128 lanes x 2 flop x clock (B200_PROFILING.md unit counts)."""
    return SM_COUNT * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.idx)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return None
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def captured_traffic(pi_kernel, workload):
    """roofline.traffic: DRAM bytes per launch of the PI kernel from the committed ncu --set full capture of THIS kernel
    on THIS workload (profiles/pi_dram_bytes_per_launch.csv: pi_kernel, workload, bytes, capture), else None."""
    tpath = os.path.join(ROOT, "profiles", "pi_dram_bytes_per_launch.csv")
    try:
        for row in open(tpath).read().splitlines()[1:]:
            f = [x.strip() for x in row.split(",")]
            if len(f) >= 3 and int(f[0]) == pi_kernel and f[1] == workload:
                return int(f[2])
    except Exception:
        pass
    return None


def make_case(cfg_index, cell_div):
    from paper_2104_00537_b200 import workloads as wl
    return wl.config(cfg_index, cell_div=cell_div)


def oracle_pass_timing(case, threads=None):
    """Time the CPU oracle as it stands: one neighbour-list build + one interaction pass."""
    import oracle
    if threads:
        oracle.set_num_threads(threads)
    st = oracle.State(case.params, case.pos, case.vel, case.rho, case.ptype)
    t0 = time.perf_counter()
    r = st.interactions(mode=1)
    dt = time.perf_counter() - t0
    return int(r["nbcount"].sum()), dt, oracle.num_threads()


def cpu_legs():
    """BASELINE.md section 3, legs B1 and B3 of the CPU baseline (B2 is the default cpu_baseline of every line): the
    oracle as it stands.  B1 = config 0, all of its 100 symplectic steps, on one core.  B3 = config 3 (periodic
    cloud), one cell-list build + one interaction pass on all cores, on the 1/8 sub-cube (126^3 sites instead of
    252^3) that BASELINE.md allows when the full pass exceeds the time budget."""
    import oracle
    from paper_2104_00537_b200 import workloads as wl
    all_threads = oracle.num_threads()
    legs = {}
    c0 = wl.config(0)
    oracle.set_num_threads(1)
    st = oracle.State(c0.params, c0.pos, c0.vel, c0.rho, c0.ptype)
    per_pass = int(st.interactions()["nbcount"].sum())
    t0 = time.perf_counter()
    st.step(c0.nsteps)
    el = time.perf_counter() - t0
    legs["B1"] = {"value": 2.0 * per_pass * c0.nsteps / el, "unit": UNIT, "cores": 1, "kind": "oracle", "wall_s": el,
                  "steps_per_s": c0.nsteps / el,
                  "sample": f"{c0.name}: all {c0.nsteps} symplectic steps ({c0.n} particles, {per_pass} interactions per "
                            f"pass counted at t=0, 2 passes per step), fp64"}
    oracle.set_num_threads(all_threads)
    c3 = wl.config(3, scale=0.5)
    ni, dt_s, cores = oracle_pass_timing(c3)
    legs["B3"] = {"value": ni / dt_s, "unit": UNIT, "cores": cores, "kind": "oracle", "wall_s": dt_s,
                  "sample": f"{c3.name} at scale 0.5 (1/8 sub-cube, {c3.n} particles): one cell-list build + one "
                            f"interaction pass, {ni} interactions, fp64"}
    return legs


def run_reference(args):
    """--impl reference: the oracle (plain C, double precision) timed on the host cores.  Each step is a
    full symplectic step on a bounded sample of the workload (config 2 geometry at scale 0.35)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2104_00537_b200 import workloads as wl
    scale = 0.35
    case = wl.config(args.config, cell_div=1, scale=scale)
    st = oracle.State(case.params, case.pos, case.vel, case.rho, case.ptype)
    per_pass = int(st.interactions()["nbcount"].sum())
    for _ in range(args.warmup):
        st.step(1)
    t0 = time.perf_counter()
    st.step(args.steps)
    el = time.perf_counter() - t0
    inter = 2.0 * per_pass * args.steps   # the dam break barely moves in a few steps: count at t=0 per pass
    value = inter / el
    cores = oracle.num_threads()
    sample = (f"config {args.config} geometry at scale {scale} ({case.n} particles, {per_pass} interactions/pass), "
              f"full symplectic steps (2 passes + update) in fp64, OpenMP over particles")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            # the arm's config is ours (tier framing); each step is a bounded sample of it, described in cpu_baseline.sample
            "config": {"workload": case.name, "sample_scale": scale, "n_particles_sample": case.n},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def aggregate_replicas(ms_local, units_local, dist=None, device="cpu"):
    """Replicas-only multi-GPU accounting: every rank runs the same workload on its own
    GPU with no data-path collective; the job's time is the MAX over ranks and its work the SUM over ranks.
    Returns (ms_max, units_total / seconds).  Works with any torch.distributed backend (nccl on GPUs, gloo in
    the CPU tests)."""
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    ms_max = float(t.item())
    return ms_max, float(u.item()) / (ms_max * 1e-3)


def run_ours(args):
    import torch
    from paper_2104_00537_b200 import sph

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cell_div = args.cell_div
    case = make_case(args.config, cell_div)
    n = case.n
    stream = torch.cuda.current_stream()
    prm = dict(case.params, integrator=1 if args.integrator == "verlet" else 0)
    compensated = args.compensated if args.compensated >= 0 else (1 if args.config == 4 else 0)
    prm["compensated_sums"] = compensated
    if args.mdbc:
        prm.update(boundary_model=1, mdbc_slip=1)
    if args.shifting:
        prm.update(shift_model=1, shift_coef=2.0, shift_fs_conc=0.85)
    S = sph.Sph(prm, pi_kernel=args.pi_kernel, count_neighbours=False, stream=stream)
    S.load_case(case)
    S.compute_interactions()
    info0 = S.get_info()
    per_pass0 = int(info0.n_interactions)

    # ---- device-resident timing: inputs already in HBM ----
    if args.develop > 0:          # advance the state before timing (the lattice order of t = 0 is the friendliest)
        S.step(args.develop)
    if args.warmup < 3 and rank == 0:
        print(f"bench.py: --warmup {args.warmup} raised to 3 (the timing rules ask for at least 3 warm-up steps)",
              file=sys.stderr)
    for _ in range(max(args.warmup, 3)):
        S.step(1)
    i0 = S.get_info()
    tm0 = S.get_timings()
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    for _ in range(args.steps):   # the timed region: per-phase profiling is OFF
        S.step(1)
    ev1.record(stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop()
    i1 = S.get_info()
    tm_mid = S.get_timings()
    inter = int(i1.n_interactions_total) - int(i0.n_interactions_total)
    launches = int(tm_mid.n_kernel_launches) - int(tm0.n_kernel_launches)
    ms_max, value = aggregate_replicas(ms_total, inter, dist, "cuda")

    # ---- second loop of the same length with the per-phase CUDA-event timers on: phase split + PI launch time ----
    S.set_profiling(True)
    for _ in range(args.steps):
        S.step(1)
    tm1 = S.get_timings()
    S.set_profiling(False)
    i2 = S.get_info()
    inter_prof = int(i2.n_interactions_total) - int(i1.n_interactions_total)
    n_pi = int(tm1.n_interaction_passes) - int(tm_mid.n_interaction_passes)

    # ---- end to end through the C ABI with host buffers (pinned): H2D + step + D2H every step ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_pos, h_vel, h_rho, h_typ = pin(case.pos), pin(case.vel), pin(case.rho), pin(case.ptype)
    o_pos = torch.empty((n, 3), dtype=torch.float64).pin_memory()
    o_vel = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    o_rho = torch.empty((n,), dtype=torch.float32).pin_memory()
    h2d = h_pos.numel() * 8 + h_vel.numel() * 4 + h_rho.numel() * 4 + h_typ.numel()
    d2h = o_pos.numel() * 8 + o_vel.numel() * 4 + o_rho.numel() * 4

    def e2e_step():
        S.load_particles_ptr(n, h_pos.data_ptr(), h_vel.data_ptr(), h_rho.data_ptr(), h_typ.data_ptr())
        S.step(1)
        S.read_fields_ptr([sph.SPH_POS, sph.SPH_VEL, sph.SPH_RHO],
                          [o_pos.data_ptr(), o_vel.data_ptr(), o_rho.data_ptr()],
                          [o_pos.numel() * 8, o_vel.numel() * 4, o_rho.numel() * 4])

    e2e_steps = max(1, min(args.steps, 5))
    e2e_step()
    ie0 = S.get_info()
    per_step_inter = int(ie0.n_interactions_total)     # counters reset at load: one step's interactions
    barrier()
    ev0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    ev1.record(stream)
    barrier()
    _, e2e_value = aggregate_replicas(ev0.elapsed_time(ev1), per_step_inter * e2e_steps, dist, "cuda")

    # ---- the same kernel on a developed state (BASELINE.json config 2 is "1000 steps"; the jittered lattice of t = 0 is
    #      the friendliest state): reload, advance, then time K more steps with the phase timers on.  Outside `value`.
    dev_steps = args.roofline_developed if args.roofline_developed >= 0 else (1000 if args.config == 2 else 0)
    developed = None
    if dev_steps > 0:             # every rank (replicas stay in step until the process group is destroyed)
        S.load_case(case)
        S.step(dev_steps)
        id0, td0 = S.get_info(), S.get_timings()
        S.set_profiling(True)
        S.step(args.steps)
        td1 = S.get_timings()
        S.set_profiling(False)
        id1 = S.get_info()
        npass = int(td1.n_interaction_passes) - int(td0.n_interaction_passes)
        developed = {"steps_before": dev_steps, "t_sim": float(id0.t), "n_out": int(id1.n_out),
                     "ms_per_launch": td1.ms_interaction / max(npass, 1),
                     "interactions_per_launch": (int(id1.n_interactions_total) - int(id0.n_interactions_total)) / max(npass, 1),
                     "ms_per_step_with_timers": sum(getattr(td1, k) for k in ("ms_key", "ms_sort", "ms_cellstart", "ms_reorder",
                                                                               "ms_interaction", "ms_dt", "ms_update",
                                                                               "ms_mdbc", "ms_shift")) / args.steps}

    if rank != 0:
        S.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (particle interaction), measured live with CUDA events ----
    peaks = measured_peaks()
    sm_max = float((clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0)
    pi_ms = (tm1.ms_interaction) / max(n_pi, 1)
    cand = CAND_PER_ACCEPTED_2D if int(case.params["dim"]) == 2 else CAND_PER_ACCEPTED
    c = cand[cell_div] if info0.pi_kernel == 1 or cell_div != 1 else cand[1]
    c = min(c, cand[1])
    flops_per_inter = FLOPS_PER_ACCEPTED + FLOPS_PER_CANDIDATE * c
    per_pass = inter_prof / max(n_pi, 1)
    achieved = per_pass * flops_per_inter / (pi_ms * 1e-3) / 1e12
    peak = fp32_peak_tflops(sm_max)
    traffic = captured_traffic(int(info0.pi_kernel), case.name)
    phases = {k: getattr(tm1, k) / args.steps for k in ("ms_key", "ms_sort", "ms_cellstart", "ms_reorder",
                                                        "ms_interaction", "ms_dt", "ms_update", "ms_mdbc", "ms_shift")}
    roofline = {"bound": "alu", "kernel": "particle interaction (a5/a6)", "achieved": achieved, "peak": peak,
                "unit": "TFLOP/s", "frac": achieved / peak,
                # accepted pairs only (41 flops each), no credit for the candidate tests
                "frac_useful": per_pass * FLOPS_PER_ACCEPTED / (pi_ms * 1e-3) / 1e12 / peak,
                "traffic": traffic,
                "peak_source": f"derived: 148 SM x 128 FP32 lanes x 2 x {sm_max:.0f} MHz; MEASURED_PEAKS.json has no FP32 figure, "
                               "the repository's own FFMA microbenchmark reaches 3.92 of 4 warp-FFMA per clock per SM = 72.9 TFLOP/s "
                               "(profiles/r2_fp32_peak.md), i.e. 98 % of this denominator",
                "flops_per_interaction": flops_per_inter, "interactions_per_launch": per_pass,
                "ms_per_launch": pi_ms, "gpips_kernel": per_pass / (pi_ms * 1e-3) / 1e9,
                "hbm_bytes_per_launch_algorithmic": 48.0 * n,
                "hbm_frac_of_measured": (48.0 * n / (pi_ms * 1e-3) / 1e9) / float(peaks.get("hbm_gbs", 6650.0))}

    if developed is not None:
        a_dev = developed["interactions_per_launch"] * flops_per_inter / (developed["ms_per_launch"] * 1e-3) / 1e12
        developed.update(achieved=a_dev, peak=peak, unit="TFLOP/s", frac=a_dev / peak,
                         gpips_kernel=developed["interactions_per_launch"] / (developed["ms_per_launch"] * 1e-3) / 1e9)

    # ---- CPU baseline: the oracle as it stands on a bounded sample (one NL build + one pass, full size) ----
    cpu = None
    if not args.no_cpu_baseline:
        try:
            ni, dt_s, cores = oracle_pass_timing(case)
            cpu = {"value": ni / dt_s, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"one cell-list build + one interaction pass (fp64) on the full {case.name} state at t=0: "
                             f"{ni} interactions in {dt_s:.2f} s"}
            assert ni == per_pass0, (ni, per_pass0)     # same neighbour pairs as the GPU found
        except AssertionError:
            raise
        except Exception as e:  # noqa: BLE001
            cpu = {"value": None, "unit": UNIT, "cores": 0, "kind": "oracle", "sample": f"failed: {e}"}
        if args.cpu_legs and cpu.get("value") is not None:
            cpu["legs"] = cpu_legs()

    ws_mb = 190.0 * n / 1e6       # particle arrays one step touches, about 190 B per particle
    if ws_mb > 126.0:
        l2_note = (f"no flush: the per-step working set (~190 B/particle x {n / 1e6:.2f} M particles = {ws_mb:.0f} MB) "
                   f"is larger than the 126 MB L2")
    else:
        l2_note = (f"NOT flushed: the per-step working set (~190 B/particle x {n / 1e6:.2f} M particles = {ws_mb:.0f} MB) "
                   f"fits the 126 MB L2, so this line is an L2-warm number")
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": case.name, "n_particles": n, "n_fluid": case.n_fluid, "n_boundary": case.n_bound,
                       "cell_div": cell_div, "pi_kernel": int(info0.pi_kernel), "integrator": args.integrator, "multi_gpu": "replicas only",
                       "boundary_model": "mdbc" if args.mdbc else "dbc", "shifting": bool(args.shifting),
                       "compensated_sums": compensated,
                       "developed_steps": args.develop + max(args.warmup, 3),
                       "warmup_requested": args.warmup,      # fewer than 3 are raised to 3 (timing rules)
                       "timing": "value: CUDA events around K steps with the per-phase timers off; phase_ms_per_step and roofline: a second loop of K steps with the timers on",
                       "l2": l2_note,
                       "interactions_per_pass_t0": per_pass0},
            "steps_per_s": args.steps / (ms_max * 1e-3),
            "gpips": value / 1e9,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps},
            "gpu_launches": launches,
            "phase_ms_per_step": phases,
            "roofline": roofline,
            "roofline_developed": developed,
            "cpu_baseline": cpu}
    print(json.dumps(line))
    S.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2 = headline)")
    ap.add_argument("--cell-div", type=int, default=1)
    ap.add_argument("--pi-kernel", type=int, default=0)
    ap.add_argument("--integrator", choices=["symplectic", "verlet"], default="symplectic",
                    help="symplectic (default, the metric's configuration) or verlet (Eq. 30-31, one pass per step)")
    ap.add_argument("--compensated", type=int, default=-1,
                    help="sph_params.compensated_sums (Kahan momentum sums, +15 %% per pass); default 1 on config 4, where the "
                         "stated tolerance needs it, else 0")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-legs", action="store_true",
                    help="also time legs B1 (config 0, 100 steps, 1 core) and B3 (config 3 sub-cube, one pass) of BASELINE.md "
                         "section 3 and print them under cpu_baseline.legs (adds about a minute of host time)")
    ap.add_argument("--roofline-developed", type=int, default=-1,
                    help="also report the interaction kernel's roofline after this many steps from t = 0 (roofline_developed; "
                         "measured after the timed region; default 1000 on config 2, 0 = off elsewhere)")
    ap.add_argument("--develop", type=int, default=0, help="advance this many steps before the warm-up and the timing")
    ap.add_argument("--mdbc", action="store_true", help="mDBC boundaries (Eq. 38-39) instead of DBC; not the metric's configuration")
    ap.add_argument("--shifting", action="store_true", help="particle shifting (Eq. 40-41, 53-54); not the metric's configuration")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
