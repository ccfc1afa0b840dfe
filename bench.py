#!/usr/bin/env python
"""bench.py -- headline benchmark of the Monte Carlo transport hot path (BASELINE.json metric:
photon packets/s and cell-crossings/s on B200; fraction of the gather-bandwidth roofline).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c1_tau1] [--impl reference]

A step = one mcrt_run_batch (transport of one batch with frozen temperatures + tally merge +
temperature update) of the workload's batch size.  Prints ONE JSON line (rank 0).
DESIGN.md section 8 states every figure's definition.
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

from paper_1201_3588_b200 import workloads as W  # noqa: E402

METRIC = "photon packets/sec"
UNIT = "packets/s"


def make_workload(name: str):
    """Bench workloads.  c1_tau1 = BASELINE.json configs[1] at tau_V = 1 (the configuration the
    10^8 packets/s target is quoted on)."""
    if name.endswith("_pah"):                                # row f2: the same workload with a transiently heated PAH
        return make_workload(name[:-4])
    if name.startswith("c1_tau"):
        return W.c1(tau_v=float(name[6:]))
    if name == "c0":
        return W.c0()
    if name == "c2":
        return W.c2()
    if name == "c3":
        return W.c3()
    if name == "c4":
        return W.c4()
    if name == "c4_256":
        return W.c4(n_root=256, batch=1 << 22)
    raise SystemExit(f"unknown workload {name}")


def describe(wl, name):
    return {"workload": name, "grid": f"{wl.n_root}^3" + (f"+{wl.n_ref}x{wl.sub}^3" if wl.n_ref else ""),
            "leaf_slots": wl.leaf_slots, "n_bins": wl.n_bins, "batch_packets": wl.batch,
            "n_sources": len(wl.sources), "seed": wl.seed}


# ---------------------------------------------------------------------------------------------
# clocks (profiling recipe: sample nvidia-smi DURING the timed region)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def wait_first(self, timeout=8.0):
        t0 = time.time()
        while self.proc is not None and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.02)

    def stop(self, t_from=0.0, t_to=float("inf")):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], [], set()
        for t, r in self.rows:
            if len(r) < 6 or t < t_from or t > t_to:
                continue
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except ValueError:
                continue
            for name, v in zip(self.NAMES, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def ncu_capture(name):
    """What the committed ncu --set full capture of this workload says about one k_transport_u launch
    (profiles/traffic.json): DRAM bytes, warp instructions, lanes per instruction; {} if none."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        with open(p) as f:
            t = json.load(f).get(name)
        if isinstance(t, dict):
            return t
    return {}


def ncu_traffic(name):
    t = ncu_capture(name).get("bytes_per_launch")
    return float(t) if t else None


def issue_peak():
    """Issue-slot ceiling of the GPU in warp instructions per second: SMs x 4 warp schedulers x 1
    instruction per clock x the maximum SM clock (B200_PROFILING.md: 148 SMs, 1965 MHz)."""
    mhz = 1965.0
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            mhz = float(json.load(f).get("sm_max_mhz", mhz))
    return 148 * 4 * mhz * 1e6


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------
# CPU oracle legs
# ---------------------------------------------------------------------------------------------
def _oracle_sample(O, wl, threads, target_seconds, n_batches=4):
    """Time the oracle, as it stands, on packets 0..n-1 of the workload in n_batches equal batches
    (temperatures update in between, as in the method) with `threads` OpenMP threads."""
    orc = O.Oracle(wl)
    probe, dt = 1024, 0.0
    while dt < 0.4 and probe < (1 << 28):                    # calibrate the sample size
        probe *= 2
        t0 = time.perf_counter()
        orc.run_batch(wl.seed, 0, probe, threads)
        dt = max(time.perf_counter() - t0, 1e-4)
    n = int(min(max(probe * target_seconds / dt, 4 * probe), 1 << 31))       # ids may run past the config's count
    per = max(n // n_batches, 1)
    orc = O.Oracle(wl)
    t0 = time.perf_counter()
    done = 0
    for _ in range(n_batches):
        orc.run_batch(wl.seed, done, per, threads)
        done += per
    dt = time.perf_counter() - t0
    c = orc.counters()
    return done / dt, c["crossings"] / dt, f"packets 0..{done - 1} in {n_batches} batches of {per} ({dt:.1f} s wall)"


def oracle_rate(wl, target_seconds=15.0):
    """cpu_baseline: the fp64 oracle on ONE core (the headline CPU figure) and on
    all host cores (OpenMP over packets), each on a bounded sample of the same workload."""
    from oracle import oracle as O
    O.build()
    cores = O.max_threads()
    v1, x1, s1 = _oracle_sample(O, wl, 1, 0.4 * target_seconds)
    vn, xn, sn = _oracle_sample(O, wl, cores, 0.6 * target_seconds)
    return {"value": vn, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": sn + ", OpenMP over packets", "crossings_per_s": xn,
            "one_core": {"value": v1, "unit": UNIT, "cores": 1, "crossings_per_s": x1, "sample": s1}}


def run_reference(args, wl, name):
    """--impl reference: the fp64 oracle on the host cores; a step = a bounded sample batch."""
    from oracle import oracle as O
    O.build()
    cores = O.max_threads()
    orc = O.Oracle(wl)
    probe, dt = 2048, 0.0
    while dt < 0.5 and probe < wl.n_packets:
        probe *= 2
        t0 = time.perf_counter()
        orc.run_batch(wl.seed, 0, probe)
        dt = max(time.perf_counter() - t0, 1e-4)
    rate = probe / dt
    budget = 120.0 / max(args.steps + args.warmup, 1)
    per = int(min(max(rate * min(budget, 10.0), 1024), wl.batch))
    orc = O.Oracle(wl)
    first = 0
    for _ in range(args.warmup):
        orc.run_batch(wl.seed, first, per)
        first += per
    c0 = orc.counters()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.run_batch(wl.seed, first, per)
        first += per
    dt = time.perf_counter() - t0
    c1 = orc.counters()
    value = args.steps * per / dt
    sample = f"{args.steps} steps of {per} packets (bounded sample of the {wl.batch}-packet batch)"
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": describe(wl, name),
           "crossings_per_s": (c1["crossings"] - c0["crossings"]) / dt,
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ---------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------
L2_BYTES = 126 << 20


def algorithmic_bytes(wl, d_cross, d_abs):
    """SURVEY.md 8(d) / DESIGN.md section 7: 4 B per crossing (density gather; the refined-cube
    marker shares that array, the descent into a refined cube costs a second 4-B gather which
    is counted as a crossing of 8 B only on two-level grids), per absorption 4 B temperature
    gather + 8 B tally read-modify-write + ceil(log2 n_bins) * 4 B of CDF probes."""
    per_cross = 8 if wl.n_ref else 4
    per_abs = 4 + 8 + 4 * int(np.ceil(np.log2(wl.n_bins)))
    return d_cross * per_cross + d_abs * per_abs, per_cross, per_abs


def time_steps(torch, ctx, wl, runner, stream, world, steps, warmup, flush, barrier):
    """`warmup` untimed + `steps` timed batches of wl.batch packages per rank.  Returns per-step CUDA
    event times (ms), the kernel times recorded inside the library, counter deltas, launches."""
    batch = wl.batch
    step_no = [0]

    def one_step():
        runner.run_batch(wl.seed, step_no[0] * world * batch, world * batch, stream)
        step_no[0] += 1

    for _ in range(warmup):
        flush.fill_(1)
        one_step()
    barrier()
    ctx.get_batch_times()
    c_before = ctx.get_counters()
    launches_before = ctx.kernel_launches()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    t_wall = time.perf_counter()
    for a, b in ev:
        flush.fill_(1)                      # L2 flush between timed iterations (not timed)
        a.record()
        one_step()
        b.record()
    barrier()
    t_wall = time.perf_counter() - t_wall
    step_ms = [a.elapsed_time(b) for a, b in ev]
    t_tr, t_up = ctx.get_batch_times()
    c_after = ctx.get_counters()
    d = {k: c_after[k] - c_before[k] for k in ("emitted", "escaped", "absorptions", "scatterings",
                                                "flights", "crossings", "lost")}
    return dict(step_ms=step_ms, t_tr=t_tr, t_up=t_up, d=d, t_wall=t_wall,
                launches=ctx.kernel_launches() - launches_before, one_step=one_step)


# Minimum lane-instructions the method needs per unit of work (DESIGN.md section 7 derives each figure): the walk
# step is the SASS instruction count of the committed loop (29 per step + 4.5 of loop overhead per step of the PTX
# step pair, profiles/r02_summary.md; a two-level grid needs at least that much per crossing); the event figures are
# hand counts of the arithmetic each event cannot do without (Philox block, -ln, DDA set-up; HG draw + rotation;
# tally + temperature gather + 7 CDF probes + isotropic draw; emission: source CDF search + direction + start cell,
# escape tally, lane refill).  Constants of the code, not of a capture: the fraction is reproducible from the
# line's own counters.
MIN_LANE_INSTR = {"crossing": 33.5, "flight": 95.0, "scattering": 50.0, "absorption": 57.0, "packet": 70.0}


def lane_issue_peak():
    """Lane-instructions per second the GPU can issue: SMs x 4 schedulers x 32 lanes x max SM clock."""
    return issue_peak() * 32.0


def rooflines(wl, name, d, tr_s, steps, gather_peak):
    """roofline of the transport kernel, every figure from THIS run's counters and kernel times (DESIGN.md
    sections 7, 8).  `frac` is algorithmic work / live kernel time / peak:
      density array L2-resident (all but C4): bound "alu" -- the minimum lane-instructions of the method
        (MIN_LANE_INSTR x this run's crossings, flights, scatterings, absorptions, packages) against
        148 SMs x 4 schedulers x 32 lanes x sm_max_mhz;
      density array beyond the L2 (C4): bound "hbm" -- SURVEY.md 8(d)(iii) algorithmic bytes against the
        measured copy bandwidth (MEASURED_PEAKS.json).
    Inside it, always: "gather" = BASELINE.json's own metric, crossings/s against the independent-gather rate
    calibrated live at this footprint (mcrt_gather_calibrate); "hbm" and "alu" = the two algorithmic figures;
    "issue_active" = executed-instruction UTILISATION from the committed ncu capture (not a roofline fraction,
    never enters frac; stale if the kernel changed after the capture named beside it)."""
    peak, peak_src = measured_peaks()
    bytes_alg, per_cross, per_abs = algorithmic_bytes(wl, d["crossings"], d["absorptions"])
    hbm_achieved = bytes_alg / tr_s / 1e9 if tr_s > 0 else 0.0
    foot = int(wl.leaf_slots) * 4
    cap = ncu_capture(name)
    hbm = {"bound": "hbm", "achieved": hbm_achieved, "peak": peak, "unit": "GB/s",
           "frac": hbm_achieved / peak, "peak_source": peak_src,
           "algorithmic_bytes": {"per_crossing": per_cross, "per_absorption": per_abs,
                                 "per_launch": bytes_alg / steps}}
    traffic = ncu_traffic(name)
    if traffic:
        hbm["traffic_over_algorithmic"] = traffic / (bytes_alg / steps)
    work = (MIN_LANE_INSTR["crossing"] * d["crossings"] + MIN_LANE_INSTR["flight"] * d["flights"]
            + MIN_LANE_INSTR["scattering"] * d["scatterings"] + MIN_LANE_INSTR["absorption"] * d["absorptions"]
            + MIN_LANE_INSTR["packet"] * d["emitted"])
    alu_ach = work / tr_s / 1e9 if tr_s > 0 else 0.0
    alu_pk = lane_issue_peak() / 1e9
    alu = {"bound": "alu", "achieved": alu_ach, "peak": alu_pk, "unit": "G lane-instructions/s", "frac": alu_ach / alu_pk,
           "peak_source": "148 SMs x 4 warp schedulers x 32 lanes x sm_max_mhz (MEASURED_PEAKS.json, else 1965 MHz)",
           "algorithmic_work": {"min_lane_instructions_per": MIN_LANE_INSTR, "per_launch": work / steps,
                                "counters_per_launch": {k: d[k] / steps for k in ("crossings", "flights", "scatterings",
                                                                                  "absorptions", "emitted")}}}
    gather = None
    if gather_peak:
        g_ach = d["crossings"] / tr_s if tr_s > 0 else 0.0
        gather = {"footprint_bytes": foot, "peak_gathers_per_s": gather_peak, "achieved_gathers_per_s": g_ach,
                  "frac": g_ach / gather_peak,
                  "what": "BASELINE.json metric '% of gather-BW roofline': peak = independent hash-indexed 4-byte "
                          "gathers/s over an array of the density footprint at full occupancy (mcrt_gather_calibrate, "
                          "measured in this run); achieved = cell crossings/s of k_transport_u.  Above 1 the walk's "
                          "locality (bricks, grouped hand-out) lets one sector serve several crossings: no ceiling then"}
    resident = foot <= 0.75 * L2_BYTES
    head = alu if resident else hbm
    roof = {"bound": head["bound"], "kernel": "k_transport_u", "achieved": head["achieved"], "peak": head["peak"],
            "unit": head["unit"], "frac": head["frac"], "peak_source": head["peak_source"],
            "traffic": traffic, "traffic_source": cap.get("capture") if traffic else None,
            "kernel_ms": 1e3 * tr_s / steps,
            "why_this_bound": ("density array L2-resident: DRAM moves a few per cent of the algorithmic bytes, the "
                               "kernel is limited by instruction issue at 18-22 of 32 lanes (profiles/)" if resident else
                               "density array beyond the L2: the gathers' sectors come from HBM (region sweeps keep "
                               "the traffic near the algorithmic bytes)"),
            "alu": alu, "hbm": hbm, "gather": gather}
    if cap.get("warp_instructions_per_launch"):
        ipl = float(cap["warp_instructions_per_launch"])
        roof["issue_active"] = {
            "frac_of_issue_slots": (ipl / (tr_s / steps)) / issue_peak() if tr_s > 0 else 0.0,
            "warp_instructions_per_launch_from_capture": ipl,
            "lanes_per_instruction_from_capture": cap.get("lanes_per_instruction"),
            "capture": cap.get("capture"),
            "what": "utilisation (executed instructions of a committed ncu capture / this run's kernel time), "
                    "not an algorithmic fraction; never enters roofline.frac"}
    return roof, gather


def update_roofline(wl, store_slots, up_s, steps):
    """k_update_temperature: a stream over the storage slots -- reads the cumulative tally (u64) and ln rho
    (fp32), writes the temperature row (fp32): 16 B per slot against the measured copy bandwidth."""
    if not up_s or up_s <= 0:
        return None
    peak, peak_src = measured_peaks()
    ach = 16.0 * store_slots * steps / up_s / 1e9
    return {"bound": "hbm", "kernel": "k_update_temperature", "achieved": ach, "peak": peak, "unit": "GB/s",
            "frac": ach / peak, "peak_source": peak_src, "algorithmic_bytes": {"per_slot": 16, "per_launch": 16.0 * store_slots},
            "kernel_ms": 1e3 * up_s / steps}


def measure_workload(torch, mcrt, wl, name, steps, warmup, stream, flush, args, calibrate=True):
    """One entry of per_config: a fresh context, `warmup` + `steps` batches on this GPU."""
    from paper_1201_3588_b200.sharding import ShardedRunner
    ctx = mcrt.from_workload(wl)
    if name.endswith("_pah"):       # a 100-C PAH holding 5 % of the dust mass (workloads.pah_share), 128 temperature states
        pah = W.pah_share(wl, n_C=100, mass_fraction=0.05)
        ctx.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, n_Tp=128)
    runner = ShardedRunner(ctx, None)
    r = time_steps(torch, ctx, wl, runner, stream, 1, steps, warmup, flush, torch.cuda.synchronize)
    secs = float(sum(r["step_ms"])) * 1e-3
    tr_s = float(r["t_tr"].sum()) * 1e-3
    gpeak = mcrt.gather_calibrate(int(wl.leaf_slots) * 4, 1 << 30, stream)[0] if calibrate else None
    roof, gather = rooflines(wl, name, r["d"], tr_s, steps, gpeak)
    d = r["d"]
    up_s = float(r["t_up"].sum()) * 1e-3
    out = {"config": describe(wl, name), "steps": steps, "warmup": warmup,
           "packets_per_s": d["emitted"] / secs, "crossings_per_s": d["crossings"] / secs,
           "ms_per_step": 1e3 * secs / steps, "kernel_ms": 1e3 * tr_s / steps,
           "update_ms": 1e3 * up_s / steps, "lost": d["lost"],
           "crossings_per_packet": d["crossings"] / max(d["emitted"], 1),
           "bound": roof["bound"], "roofline_frac": roof["frac"],
           "alu_algorithmic_frac": roof["alu"]["frac"],
           "hbm_algorithmic_frac": roof["hbm"]["frac"],
           "gather_frac": gather["frac"] if gather else None,
           "traffic_over_algorithmic": roof["hbm"].get("traffic_over_algorithmic"),
           "update_roofline": update_roofline(wl, ctx.store_slots(), up_s, steps)}
    if name.endswith("_pah"):       # the batch-end time of a PAH run is k_pah_update (P(T) of every leaf) + k_update_temperature
        out["pah_update_ms"] = out["update_ms"]
        out["update_roofline"] = None
    ctx.destroy()
    return out


def measure_tau_sweep(torch, mcrt, repeats=3):
    """BASELINE.json configs[1] IS four independent runs (tau_V = 0.1, 1, 10, 100; 10^7 packages each in ten
    batches).  One after the other on one stream, every batch ends in a tail in which the lanes run dry (21 % of
    a launch); as four contexts on four streams the next run's blocks move into the SMs the tail frees.  Both
    ways give bit-identical tallies.  Wall clock around the 40 batches, device-synchronised, best of `repeats`."""
    wls = [W.c1(tau_v=t) for t in (0.1, 1.0, 10.0, 100.0)]

    def job(concurrent):
        ctxs = [mcrt.from_workload(w) for w in wls]
        streams = [torch.cuda.Stream() for _ in ctxs] if concurrent else [torch.cuda.current_stream()] * len(ctxs)
        for c, w, st in zip(ctxs, wls, streams):             # warm-up: one batch each, then forget it
            c.run_batch(w.seed, 0, w.batch, st.cuda_stream)
        torch.cuda.synchronize()
        for c in ctxs:
            c.reset_tallies(3)
        torch.cuda.synchronize()
        parts = [list(w.batches()) for w in wls]
        t0 = time.perf_counter()
        for i in range(len(parts[0])):
            for c, w, st, pt in zip(ctxs, wls, streams, parts):
                c.run_batch(w.seed, pt[i][0], pt[i][1], st.cuda_stream)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        res = [(c.get_counters()["escaped"], c.get_counters()["lost"], int(c.get_sed().sum()),
                int(c.get_cell_energy()[0].sum())) for c in ctxs]
        for c in ctxs:
            c.destroy()
        return dt, res
    best = {}
    ref = None
    for label, conc in (("serial", False), ("concurrent", True)):
        for _ in range(repeats):
            dt, res = job(conc)
            ref = ref or res
            if res != ref:
                return {"error": f"{label}: tallies differ from the serial run"}
            best[label] = min(best.get(label, dt), dt)
    n = sum(w.n_packets for w in wls)
    return {"packets": n, "serial_ms": 1e3 * best["serial"], "concurrent_ms": 1e3 * best["concurrent"],
            "serial_packets_per_s": n / best["serial"], "concurrent_packets_per_s": n / best["concurrent"],
            "gain": best["serial"] / best["concurrent"], "identical_tallies": True,
            "what": "configs[1] whole: 4 x 10^7 packages; four contexts on one stream vs on four streams"}


PER_CONFIG = (("c0", 6), ("c1_tau0.1", 4), ("c1_tau10", 4), ("c1_tau100", 4), ("c2", 3), ("c3", 3), ("c4", 3),
              ("c1_tau1_pah", 4), ("c2_pah", 3))


def run_gpu(args, wl, name):
    import torch
    import torch.distributed as dist
    from paper_1201_3588_b200 import build as B, mcrt

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; "
                         "use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        B.build_library()
    if world > 1:
        dist.barrier()
    mcrt.lib()

    stream = torch.cuda.current_stream().cuda_stream
    ctx = mcrt.from_workload(wl, layout=args.layout)
    if name.endswith("_pah"):                                # row f2 as the headline workload (--workload c1_tau1_pah)
        pah = W.pah_share(wl, n_C=100, mass_fraction=0.05)
        ctx.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, n_Tp=128)
    if args.threads or args.blocks_per_sm:
        ctx.set_launch(args.threads, args.blocks_per_sm)
    if args.quorum:
        ctx.set_walk_quorum(args.quorum)
    if args.source_order is not None:
        ctx.set_source_order(args.source_order)
    if args.tail_mode is not None:
        ctx.set_tail_mode(args.tail_mode)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    from paper_1201_3588_b200.sharding import ShardedRunner
    runner = ShardedRunner(ctx, dist if world > 1 else None)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_first()
    t_load0 = time.time()
    # One step = one batch of wl.batch packages per rank (weak scaling): the global batch of world*batch
    # packet ids is dealt to the ranks in contiguous ranges; N > 1 all-reduces the batch's uint32 tallies
    # before the T update (sharding.ShardedRunner).
    r = time_steps(torch, ctx, wl, runner, stream, world, args.steps, args.warmup, flush, barrier)
    step_ms, t_tr, t_up, d, launches = r["step_ms"], r["t_tr"], r["t_up"], r["d"], r["launches"]
    total_ms = float(sum(step_ms))
    # the timed region may be far shorter than nvidia-smi's sampling period: keep the same
    # load running (untimed) until the clock record holds at least ~1.5 s under load
    while time.time() - t_load0 < 1.5:
        r["one_step"]()
        torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop(t_load0, time.time()) if rank == 0 else None
    if clocks is not None:
        clocks["window"] = "warm-up + timed steps + identical untimed steps up to 1.5 s"
    stats = torch.tensor([total_ms, float(t_tr.sum()), float(t_up.sum())], dtype=torch.float64,
                         device="cuda")
    sums = torch.tensor([d["emitted"], d["crossings"], d["absorptions"], d["scatterings"],
                         d["lost"], launches], dtype=torch.int64, device="cuda")
    if world > 1:
        dist.all_reduce(stats, op=dist.ReduceOp.MAX)
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)
    total_ms, tr_ms, up_ms = [float(v) for v in stats.cpu()]
    n_emit, n_cross, n_abs, n_sca, n_lost, launches = [int(v) for v in sums.cpu()]

    # ---- e2e: a whole user job from HOST buffers to HOST results -------
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(args, wl, mcrt, torch, dist, rank, world, stream)

    # ---- gather roofline: independent 4-byte gathers over the density
    # footprint of this workload, measured live by the library's calibration kernel ----------
    gpeak = None
    if rank == 0 and not args.no_gather:
        gpeak = mcrt.gather_calibrate(int(wl.leaf_slots) * 4, 1 << 31, stream)[0]

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    secs = total_ms * 1e-3
    store_slots = ctx.store_slots()
    ctx.destroy()
    tr_s = float(t_tr.sum()) * 1e-3                          # dominant kernel: this rank's launches
    roof, gather = rooflines(wl, name, d, tr_s, args.steps, gpeak)
    roof["kernel_share_of_step"] = tr_s / (float(sum(step_ms)) * 1e-3)
    out = {"metric": METRIC, "value": n_emit / secs, "unit": UNIT, "n_gpus": world,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
           "data": "synthetic",
           "config": dict(describe(wl, name), l2="flushed between timed steps (256 MiB write)",
                          parallelism=f"packet-sharded x{world}",
                          launch=f"{ctx_launch_desc(args)}"),
           "crossings_per_s": n_cross / secs,
           "per_packet": {"crossings": n_cross / max(n_emit, 1), "absorptions": n_abs / max(n_emit, 1),
                          "scatterings": n_sca / max(n_emit, 1)},
           "lost": n_lost,
           "kernel_ms_per_step": {"transport": tr_ms / args.steps, "temperature_update": up_ms / args.steps},
           "wall_ms_per_step_incl_flush": 1e3 * r["t_wall"] / args.steps,
           "roofline": roof, "gpu_launches": launches, "clocks": clocks}
    out["update_roofline"] = update_roofline(wl, store_slots, up_ms * 1e-3, args.steps)
    if e2e is not None:
        out["e2e"] = e2e
    # ---- every other config of BASELINE.json, at reduced step counts, in the same invocation ----
    if world == 1 and not args.no_per_config:
        per = {name: {k: v for k, v in (("packets_per_s", out["value"]), ("crossings_per_s", out["crossings_per_s"]),
                                         ("ms_per_step", out["ms_per_step"]),
                                         ("kernel_ms", roof["kernel_ms"]), ("bound", roof["bound"]),
                                         ("roofline_frac", roof["frac"]),
                                         ("alu_algorithmic_frac", roof["alu"]["frac"]),
                                         ("hbm_algorithmic_frac", roof["hbm"]["frac"]),
                                         ("gather_frac", gather["frac"] if gather else None), ("lost", n_lost))}}
        for wname, wsteps in PER_CONFIG:
            if wname == name:
                continue
            try:
                per[wname] = measure_workload(torch, mcrt, make_workload(wname), wname, wsteps, 3, stream, flush, args)
            except Exception as e:                           # a config that cannot run must not hide the others
                per[wname] = {"error": f"{type(e).__name__}: {e}"}
            torch.cuda.empty_cache()
        out["per_config"] = per
        try:
            out["c1_tau_sweep"] = measure_tau_sweep(torch, mcrt)
        except Exception as e:
            out["c1_tau_sweep"] = {"error": f"{type(e).__name__}: {e}"}
    if not args.no_cpu and world >= 1:
        out["cpu_baseline"] = oracle_rate(wl, target_seconds=args.cpu_seconds)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def ctx_launch_desc(args):
    return (f"threads={args.threads or 'default'} blocks_per_sm={args.blocks_per_sm or 'default'} "
            f"quorum={args.quorum or 'auto'} layout={args.layout or 'auto'}")


def run_e2e_job(args, wl, mcrt, torch, dist, rank, world, stream):
    """End to end through the public API with HOST buffers: the job starts from host arrays
    (grid_create/set_opacity/set_source copy them H2D inside the timed region) and every step
    ends with a device->host read of that step's results (SED, counters, cell energies, cell
    temperatures) into pinned host buffers.  The read-out of batch k is queued behind it
    (mcrt_results_begin) and overlaps batch k+1; it is waited for before its buffers are reused.
    Value = packets of all steps / wall time, device-synchronised, max over ranks."""
    batch = wl.batch
    rho = torch.from_numpy(np.ascontiguousarray(wl.rho_root)).pin_memory().numpy()
    steps = args.warmup + args.steps
    slots = wl.leaf_slots
    pin = lambda shape, dt: torch.empty(shape, dtype=dt).pin_memory().numpy()
    mk = lambda: dict(n_abs=pin((slots,), torch.int64).view(np.uint64), T=pin((slots,), torch.float32),
                      sed=pin((3, wl.n_bins), torch.int64).view(np.uint64),
                      emitted_per_bin=pin((wl.n_bins,), torch.int64).view(np.uint64))
    bufs = [mk(), mk()]                                      # allocated once, reused every other step
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    ctx = mcrt.Context()
    ctx.grid_create(wl.n_root, wl.sub, wl.origin, wl.root_size, wl.refine, rho, wl.rho_sub)
    ctx.set_opacity(wl.lambda_edges_um, wl.weight, wl.kabs, wl.ksca, wl.g)
    ctx.set_source(wl.sources)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    from paper_1201_3588_b200.sharding import ShardedRunner
    runner = ShardedRunner(ctx, dist if world > 1 else None)
    pending, n_read = None, 0
    for s in range(steps):
        runner.run_batch(wl.seed, s * world * batch, world * batch, stream)
        h = ctx.results_begin(bufs[s % 2])
        if pending is not None:
            n_read += ctx.results_wait(pending)["counters"]["emitted"] > 0
        pending = h
    last = ctx.results_wait(pending)
    n_read += 1
    torch.cuda.synchronize()
    dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(dt, op=dist.ReduceOp.MAX)
    dt = float(dt.cpu())
    assert n_read == steps and last["counters"]["emitted"] > 0
    d2h = sum(v.nbytes for v in bufs[0].values()) + 7 * 8
    h2d_job = wl.rho_root.nbytes + (0 if wl.rho_sub is None else wl.rho_sub.nbytes) \
        + (0 if wl.refine is None else wl.refine.nbytes + 4 * wl.refine.size) \
        + wl.kabs.nbytes * 3 + wl.lambda_edges_um.nbytes
    ctx.destroy()
    return {"value": steps * batch * world / dt, "unit": UNIT,
            "h2d_bytes_per_step": h2d_job / steps, "d2h_bytes_per_step": d2h,
            "job_ms": 1e3 * dt, "setup_ms": 1e3 * t_setup, "steps_ms": 1e3 * (dt - t_setup),
            "value_steps_only": steps * batch * world / (dt - t_setup),
            "what": f"one job of {steps} batches from host arrays: grid/opacity/source set-up "
                    "(H2D) + run_batch + host read-back of SED, counters, cell energy and "
                    "temperature after EVERY batch (pinned buffers; the read-out of batch k "
                    "overlaps batch k+1); wall clock, device-synchronised"}


def run_e2e(args, wl, mcrt, torch, dist, rank, world, stream, repeats=3):
    """The whole job `repeats` times, each from scratch (new context, host arrays in, host results out); the
    MEDIAN job is reported and every job's wall time is listed.  A ~10 ms job timed by wall clock once is at the
    mercy of one slow cudaMalloc / cudaMallocHost (jobs of 13, 33 and 145 ms were seen back to back)."""
    jobs = [run_e2e_job(args, wl, mcrt, torch, dist, rank, world, stream) for _ in range(repeats)]
    order = sorted(range(repeats), key=lambda i: jobs[i]["job_ms"])
    out = dict(jobs[order[repeats // 2]])
    out["job_ms_all"] = [j["job_ms"] for j in jobs]
    out["cold_first_job"] = {"value": jobs[0]["value"], "job_ms": jobs[0]["job_ms"], "setup_ms": jobs[0]["setup_ms"],
                             "what": "the first of the jobs: its device blocks are not all in the library's cache yet "
                                     "(only those the benchmark's own context of the same shape gave back)"}
    out["what"] += (f"; the job is run {repeats} times, each with a new context from host arrays; the MEDIAN job is "
                    "reported: a WARM-POOL job -- the library caches the device blocks a destroyed context gives back "
                    "(mcrt_release_cached_memory frees them), so jobs 2 and 3 allocate nothing; cold_first_job is the first")
    return out


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` without a launcher: start N ranks on this node ourselves."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                     # the communicator log shows the ranks (and NVLS)
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    raise SystemExit(subprocess.call(cmd, env=env))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--workload", default="c1_tau1")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--quorum", type=int, default=0, help="walk-loop quorum (0 = automatic)")
    ap.add_argument("--source-order", type=int, default=None,
                    help="hand packages out grouped by source: 1 on, 0 off (default: automatic)")
    ap.add_argument("--tail-mode", type=int, default=None, help="end of a batch: -1 auto; bit 0: quorum follows the live lanes; bit 1: temperature update fused into the transport launch")
    ap.add_argument("--layout", type=int, default=0, help="0 auto, 1 x-fastest, 2 bricked")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-gather", action="store_true", help="skip the gather-roofline calibration")
    ap.add_argument("--no-per-config", action="store_true", help="skip the other configs (per_config)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "native" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        if rank != 0:
            return
        run_reference(args, make_workload(args.workload), args.workload)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)
    if args.gpus != int(os.environ.get("WORLD_SIZE", "1")):
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE', '1')}")
    run_gpu(args, make_workload(args.workload), args.workload)


if __name__ == "__main__":
    main()
