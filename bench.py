#!/usr/bin/env python
"""bench.py — proton histories/s of the full-physics hot path (pmc_simulate) on config C4, with roofline,
end-to-end (host-buffer) throughput and the fp64 CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4|c1|c3_150|c5]

One "step" = one pmc_simulate call: the whole hot path (spot sampler, condensed-history transport, elastic, INC,
evaporation, 10-batch statistics) over `--histories` primaries (default: the workload's own count, 1e7 for C4).
N > 1 (torchrun, one rank per GPU): weak scaling, every rank simulates the same number of histories with
disjoint global history ids; the per-rank doses are combined with one NCCL all-reduce per step.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "proton histories/sec (full physics, dose on CT grid)"
UNIT = "histories/s"
# DESIGN.md section 7 "Roofline": algorithmic thread-instructions of ONE condensed-history step of the step kernel, item by
# item - what the method itself needs with ideal code (every multiply-add fused, no moves, no address arithmetic, no
# reconvergence instructions), counted against the SASS of profiles/r02_transport_sass_histogram.md.
ALGO_ITEMS = {
    "philox4x32_10_two_blocks (2 x 10 rounds x (2 mul.wide + 2 xor3))": 80,
    "seven_uniforms_to_float (2 each)": 14,
    "hu_gather_bin_lookup_density": 8,
    "ln_E_and_table_index": 8,
    "sigma_lerp_and_nuclear_distance (ln u, 1/Sigma)": 8,
    "range_spline_and_exp (4 loads, 9 flops, ex2)": 15,
    "face_distances_two_calls (3 axes x 6 + min/argmin)": 42,
    "step_length_min_of_four": 8,
    "hinge_move_highland_rayleigh (rcp, lg2 x 2, sqrt)": 15,
    "sincos_theta_series_and_azimuth": 15,
    "direction_rotation_and_renormalisation": 24,
    "second_leg_position_clamps_axis": 15,
    "mean_loss (log1p, inverse spline, expm1)": 36,
    "straggling (kinematics 14, normal 7, T_c/mu/mean 12, Poisson 8, two candidates 14, cumulants 12, Wilson-Hilferty 12, clamp 2)": 81,
    "energy_update_and_termination": 8,
    "voxel_index_update_and_bounds": 12,
    "dose_red (address, atomic)": 4,
    "loop_vote_refill_check": 10,
}
ALGO_INST_PER_STEP = float(sum(ALGO_ITEMS.values()))
# One-off `ncu --set full` capture of the first-generation step-kernel launch of a 1e7-history C4 step
# (profiles/r02_transport_full.md; NOT measured in this run): DRAM bytes per history, executed thread-instructions per
# condensed step, active lanes per warp instruction, issue-slot utilisation.
NCU_CAPTURE = {"source": "profiles/r02_transport_full.md, profiles/r03_transport_pipes.md, profiles/r03_c5_transport.md (one-off ncu "
                         "captures at head c17c33c, step kernel unchanged since r02: 2.9848e10 warp instructions in both; not "
                         "measured in this run)",
               "dram_bytes_per_history_c4": 79.3, "executed_thread_inst_per_step": 634.0, "lanes_per_warp_inst": 29.2,
               "issue_slot_utilisation_pct": 81.6,
               # which pipe binds (r03): none - the busiest pipe is the ALU at 56 % of its issue rate, the MUFU (XU) pipe 42 %,
               # FMA heavy / lite 40 / 37 %; the kernel is bound by the issue slots themselves (81.6 % busy)
               "binding": "issue slots", "pipe_pct_of_peak": {"alu": 56.4, "xu": 42.4, "fmaheavy": 40.5, "fmalite": 37.4,
                                                              "adu": 24.1, "lsu": 10.2, "cbu": 3.9, "uniform": 0.5},
               "dram_bytes_per_history_c5": 68.6, "c5_l2_hit_rate_pct": 70.1, "c5_issue_slot_utilisation_pct": 82.2}
ISSUE_LANES_PER_SM_PER_CLK = 128.0     # 4 schedulers x 32 lanes
N_SM = 148


def _env_int(k, d):
    try:
        return int(os.environ.get(k, d))
    except ValueError:
        return d


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def _cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def time_oracle(w, tables, target_s, seed):
    """The oracle as it stands on the host cores, on a bounded sample of the workload -> (hist/s, n, seconds)."""
    from oracle import Oracle
    o = Oracle(tables, w["materials"])
    o.load_ct(w["hu"], w["vox"])
    n = 20000
    t0 = time.perf_counter(); o.simulate(w["spots"], n, seed); dt = time.perf_counter() - t0
    rate = n / dt
    n2 = int(min(max(rate * target_s, 20000), 5_000_000))
    if n2 > 2 * n:
        t0 = time.perf_counter(); o.simulate(w["spots"], n2, seed + 1); dt = time.perf_counter() - t0
        n = n2
    return n / dt, n, dt


def run_reference(args, rank):
    """--impl reference: the fp64 oracle on the host cores, bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    import inputs
    w = inputs.workload(args.workload)
    tables = inputs.make_physics_tables()
    from oracle import Oracle
    o = Oracle(tables, w["materials"]); o.load_ct(w["hu"], w["vox"])
    n = 20000
    t0 = time.perf_counter(); o.simulate(w["spots"], n, 1000); dt = time.perf_counter() - t0
    budget = 150.0 / max(1, args.steps + args.warmup)
    n_step = int(min(max(n / dt * min(budget, 20.0), 5000), 2_000_000))
    for i in range(args.warmup):
        o.simulate(w["spots"], n_step, 2000 + i)
    t0 = time.perf_counter()
    for i in range(args.steps):
        o.simulate(w["spots"], n_step, 3000 + i)
    dt = time.perf_counter() - t0
    v = n_step * args.steps / dt
    sample = f"{n_step} histories of {w['name']} per step (of {w['n_histories']})"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["label"], "histories_per_step": n_step, "n_spots": w["n_spots"]},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": _cores(), "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--histories", type=int, default=0, help="histories per step and per rank (0 = the workload's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--option", action="append", default=[], metavar="KEY=VALUE",
                    help="pmc_set_option before the run (e.g. dose_aggregate=1, dose_scoring=0, n_batches=40)")
    ap.add_argument("--no-extras", action="store_true", help="skip the C2 / C5 / LET_d / gamma-index measurements")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    rank, local_rank, world = _env_int("RANK", 0), _env_int("LOCAL_RANK", 0), _env_int("WORLD_SIZE", 1)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    import inputs
    from paper_1409_8336_b200 import Pmc
    from paper_1409_8336_b200.sharding import weak_shard, combine_dose

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    w = inputs.workload(args.workload)
    tables = inputs.make_physics_tables()
    n_hist = args.histories or w["n_histories"]
    stream = torch.cuda.Stream(device=dev)
    pm = Pmc(local_rank, stream=stream)
    pm.load_physics_tables(tables)
    pm.set_hu_materials(w["materials"])
    hu_dev = torch.as_tensor(w["hu"], device=dev)
    pm.load_ct(hu_dev, w["vox"])
    offset, _ = weak_shard(n_hist, rank)
    pm.set_option("history_offset", float(offset))
    n_batches = int(tables["n_batches"])            # what the context runs with: the tables' value unless an option sets it
    for kv in args.option:
        k_, v_ = kv.split("=", 1)
        pm.set_option(k_, float(v_))
        if k_ == "n_batches":
            n_batches = int(float(v_))
    spots = w["spots"]
    nvox = int(w["hu"].size)
    dose = torch.empty(w["hu"].shape, dtype=torch.float32, device=dev)
    sigma = torch.empty_like(dose)
    l2_flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def step(i):
        pm.simulate(spots, n_hist, w["seed"] + i, out=(dose, sigma))
        if world > 1:
            with torch.cuda.stream(stream):
                combine_dose(dose, sigma, n_hist)

    for i in range(args.warmup):
        step(i)
    barrier()

    # ---- device-resident timing: K steps, CUDA events on the library's stream, L2 flushed between steps
    sampler = ClockSampler(local_rank); sampler.start()
    time.sleep(0.3)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_transport = 0.0; n_transport = 0; launches = 0; steps_total = 0
    klass = {k: 0.0 for k in ("sampler_ms", "transport_ms", "elastic_ms", "inc_ms", "evaporation_ms", "statistics_ms")}
    cnt_last = None
    barrier()
    for i in range(args.steps):
        with torch.cuda.stream(stream):
            l2_flush.fill_(i & 0xFF)
        ev[i][0].record(stream)
        step(args.warmup + i)
        ev[i][1].record(stream)
        tm, cnt_last = pm.timing(), pm.counters()
        t_transport += tm["transport_ms"]; n_transport += tm["launches_transport"]; launches += tm["launches_total"]
        steps_total += cnt_last["n_steps"]
        for k in klass:
            klass[k] += tm[k]
    barrier()
    clocks = sampler.stop()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    value = world * n_hist * args.steps / (ms * 1e-3)

    # ---- end to end through the C-ABI with HOST buffers: HU grid + spots host->device, dose + sigma device->host
    hu_pin = torch.as_tensor(w["hu"]).pin_memory()
    dose_h = torch.empty(w["hu"].shape, dtype=torch.float32).pin_memory()
    sigma_h = torch.empty_like(dose_h).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))
    pm.load_ct(hu_pin.numpy(), w["vox"]); pm.simulate_host(spots, n_hist, 99, dose_h.numpy(), sigma_h.numpy())   # warm
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        pm.load_ct(hu_pin.numpy(), w["vox"])
        pm.simulate_host(spots, n_hist, w["seed"] + 100 + i, dose_h.numpy(), sigma_h.numpy())
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_value = world * n_hist * e2e_steps / float(t.item())
    h2d = int(w["hu"].nbytes + spots.nbytes)
    d2h = int(2 * nvox * 4)

    # ---- other rows of SURVEY 8(d)/(f), measured after the timed steps on rank 0 (not part of `value`)
    extras = None
    if rank == 0 and not args.no_extras:
        extras = measure_extras(pm, w, n_hist, spots, hu_dev, stream, dev, tables)

    if rank == 0:
        # ---- roofline of the dominant kernel (transport_kernel): plain-ALU issue bound
        sm_mhz = clocks["sm_mhz"] or 1965.0
        peak = N_SM * ISSUE_LANES_PER_SM_PER_CLK * sm_mhz * 1e6 / 1e9            # G thread-inst/s at the clock seen
        achieved = ALGO_INST_PER_STEP * steps_total / (t_transport * 1e-3) / 1e9 if t_transport > 0 else 0.0
        roofline = {"bound": "alu", "kernel": "transport_kernel", "achieved": achieved, "peak": peak,
                    "unit": "Gthread-inst/s", "frac": achieved / peak if peak else None,
                    "traffic": NCU_CAPTURE["dram_bytes_per_history_c4"] * n_hist if w["name"] == "c4" else None,
                    "traffic_note": "from a one-off ncu capture (DRAM bytes of the first-generation launch), not measured "
                                    "in this run; the kernel is issue-bound, HBM carries < 1 % of its peak",
                    "ncu_capture": NCU_CAPTURE,
                    "frac_of_executed": (NCU_CAPTURE["executed_thread_inst_per_step"] * steps_total / (t_transport * 1e-3) / 1e9
                                         / peak) if (t_transport > 0 and peak and w["name"] == "c4") else None,
                    "algorithmic_items": ALGO_ITEMS,
                    "peak_source": "148 SMs x 4 schedulers x 32 lanes x median SM clock under load (derived, DESIGN.md)",
                    "avg_launch_ms": t_transport / max(1, n_transport), "launches": n_transport,
                    "algorithmic_inst_per_condensed_step": ALGO_INST_PER_STEP,
                    "condensed_steps_per_history": steps_total / (n_hist * args.steps),
                    "kernel_share_of_step": t_transport / ms if ms else None,
                    "hbm_gbs_peak_measured": _measured_hbm()}
        cpu = None
        if not args.no_cpu_baseline:
            v, n_s, dt = time_oracle(w, tables, args.cpu_seconds, 777)
            cpu = {"value": v, "unit": UNIT, "cores": _cores(), "kind": "oracle",
                   "sample": f"{n_s} histories of {w['name']} ({dt:.1f} s, OpenMP over histories, fp64)"}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w["label"], "histories_per_step_per_gpu": n_hist, "n_spots": w["n_spots"],
                       "n_batches": n_batches, "l2": "flushed between timed steps (256 MiB write)",
                       "parallelism": f"history-sharded x{world}", "options": args.option},
            "clocks": {k: clocks[k] for k in ("sm_mhz", "sm_max_mhz", "reasons")},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps},
            "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu, "extras": extras,
            "kernel_ms_per_step": {k: v / args.steps for k, v in klass.items()},
            "counters_last_step": {k: cnt_last[k] for k in ("n_steps", "n_elastic", "n_nonelastic",
                                                            "n_secondary_protons", "n_generations", "n_missed", "n_host_waits")},
            "context": "paper: ~20 s per 1e7 histories on a GTX680 incl. transfers (PAPER.md:L15), i.e. ~5e5 hist/s",
        }
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def measure_extras(pm, w, n_hist, spots, hu_dev, stream, dev, tables):
    """LET_d and gamma index on the bench workload; pmc_nonelastic events/s on the paper's Table I workload (C2,
    PAPER.md:L187-203: 2.6e6 events, p + 16O and p + 40Ca at 200 MeV, records copied to the host); C5 histories/s."""
    import torch
    import inputs
    out = {}
    pm.load_ct(hu_dev, w["vox"])
    pm.set_option("score_letd", 1.0)
    pm.simulate(spots, n_hist, w["seed"] + 200)
    d_a, _ = pm.simulate(spots, n_hist, w["seed"] + 201); let_ms = pm.timing()["total_ms"]; d_a = d_a.clone()
    pm.set_option("score_letd", 0.0)
    d_b, _ = pm.simulate(spots, n_hist, w["seed"] + 202); plain_ms = pm.timing()["total_ms"]
    with torch.cuda.stream(stream):                      # the library launches on `stream`: mask and time there too
        tissue = torch.as_tensor(w["hu"] >= -950, device=dev)
        d_a = d_a * tissue; d_b = d_b * tissue
    stream.synchronize()
    pm.gamma_index(d_a, d_b, w["vox"], 0.02, 0.2, 0.1)
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(stream)
    for _ in range(5):
        _, g_rate = pm.gamma_index(d_a, d_b, w["vox"], 0.02, 0.2, 0.1)
    g1.record(stream); stream.synchronize()
    out.update(letd_scoring_ms_per_step=let_ms, same_without_letd_ms=plain_ms,
               gamma_index_2pct_2mm_ms_per_call=g0.elapsed_time(g1) / 5, gamma_pass_rate_two_seeds=g_rate)
    # C2: standalone non-elastic collisions
    c2 = {}
    n_ev = 2_600_000
    pm.nonelastic(8, 16, 200.0, 10_000, 1)
    for name, (z, a) in (("p+16O_200MeV", (8, 16)), ("p+40Ca_200MeV", (20, 40))):
        t0 = time.perf_counter(); rec, off = pm.nonelastic(z, a, 200.0, n_ev, 7); dt = time.perf_counter() - t0
        cn = pm.counters()
        c2[name] = {"events_per_s": n_ev / dt, "events": n_ev, "records": int(len(rec)), "seconds_incl_copy_to_host": dt,
                    "inc_tries_per_event": cn["n_inc_tries"] / n_ev, "guard_trips": cn["n_inc_guard_trips"],
                    "capacity_trips": cn["n_inc_cap_trips"], "max_stack": cn["inc_max_stack"], "max_out": cn["inc_max_out"]}
        del rec, off
    c2["context"] = "paper Table I (GTX680, fast-math): 3.9e5 (16O) and 2.7e5 (40Ca) events/s"
    out["c2_pmc_nonelastic"] = c2
    # C5: the large pelvis case, all 1e8 histories once (after a short warm-up)
    w5 = inputs.workload("c5")
    pm.set_hu_materials(w5["materials"])
    hu5 = torch.as_tensor(w5["hu"], device=dev)
    pm.load_ct(hu5, w5["vox"])
    pm.simulate(w5["spots"], 1_000_000, 1)
    t0 = time.perf_counter(); pm.simulate(w5["spots"], w5["n_histories"], w5["seed"]); dt = time.perf_counter() - t0
    tm, cn = pm.timing(), pm.counters()
    out["c5"] = {"workload": w5["label"], "histories_per_s": w5["n_histories"] / (tm["total_ms"] * 1e-3),
                 "ms_device": tm["total_ms"], "seconds_wall": dt, "steps_per_history": cn["n_steps"] / w5["n_histories"],
                 "kernel_ms": {k: tm[k] for k in ("sampler_ms", "transport_ms", "elastic_ms", "inc_ms", "evaporation_ms",
                                                  "statistics_ms")}, "n_spots": w5["n_spots"]}
    # C5's own roofline block (same plain-ALU issue bound as C4: profiles/r03_c5_transport.md shows 82 % issue-slot
    # utilisation, 70 % L2 hit rate and 0.2 % of the HBM peak although its 2.1 GB of tallies do not fit the L2)
    peak5 = N_SM * ISSUE_LANES_PER_SM_PER_CLK * 1965.0e6 / 1e9
    ach5 = ALGO_INST_PER_STEP * cn["n_steps"] / (tm["transport_ms"] * 1e-3) / 1e9 if tm["transport_ms"] > 0 else 0.0
    out["c5"]["roofline"] = {"bound": "alu", "kernel": "transport_kernel", "achieved": ach5, "peak": peak5,
                             "unit": "Gthread-inst/s", "frac": ach5 / peak5, "peak_source": "148 SMs x 128 lanes x 1965 MHz (nominal; "
                             "the main line uses the clock sampled under load)",
                             "traffic": NCU_CAPTURE["dram_bytes_per_history_c5"] * w5["n_histories"],
                             "traffic_note": "DRAM bytes of a first-generation launch from the one-off capture, per history x histories"}
    pm.set_hu_materials(w["materials"]); pm.load_ct(hu_dev, w["vox"])
    return out


def _measured_hbm():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f).get("hbm_gbs")
    except (OSError, ValueError):
        return None


if __name__ == "__main__":
    main()
