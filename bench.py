#!/usr/bin/env python
"""Benchmark of the tracking hot path (contract: see the task statement / DESIGN.md section 8).

A step = one pass of the whole hot path over one batch: restore the seeded synthetic
ensemble (device copy), then ``xt_track`` it for the config's number of turns through the
config's lattice.  Default workload: BASELINE.json configs[3] (LHC-sized lattice with
misalignments, 10^7 particles, 100 turns, SoA FP64 ~1 GB).  ``value`` is
particle*element*turns/s over all ranks with inputs resident in HBM; ``e2e`` is the same
metric through ``xt_track_host`` with pinned HOST buffers (H2D + D2H inside the timed
region).  The roofline is the FP64 ALU pipe: peak = the library's own DFMA microbenchmark
measured in this run.

``value`` counts the element visits of particles that were still alive (completed turns only,
SURVEY.md 8(d)); ``nominal_value`` counts n_part x n_elem x n_turns.  ``also`` is configs[2], the other
configuration the target names, timed in the same run as the mean over >= 5 steps with its own
roofline.  ``--config 4`` is the survival study (compaction every 1000 turns, a few thousand turns by
default) and adds the timing of the compaction passes against the measured HBM peak.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from xt_inputs import configs as C  # noqa: E402

METRIC = "particle*element*turns/s (FP64)"
UNIT = "particle*element*turns/s"
WORKLOADS = {
    2: "configs[2]: synthetic LHC-sized ring, 8606 elements (order-15 multipole errors, elliptical "
       "apertures, 8 cavities), 100000 particles (6D Gaussian 1 sigma), 1000 turns",
    3: "configs[3]: LHC-sized ring with SRotation/XYShift misalignments, 10366 elements, "
       "10000000 particles (6D Gaussian 2 sigma, SoA FP64 ~1 GB), 100 turns",
    1: "configs[1]: FODO ring with sextupoles and rectangular apertures, 71 elements, 1000000 "
       "particles (polar grid), 1000 turns",
    0: "configs[0]: thin-lens FODO ring, 41 elements, 1000 particles, 100 turns",
    4: "configs[4]: dynamic-aperture survival study on the LHC-sized ring with strong octupoles, 8606 "
       "elements, 2000400 particles (polar grid x 6 momentum offsets), compaction every 1000 turns, "
       "survival histogram; bench runs --turns of the 100000 (default 3000)",
}
BENCH_TURNS = {4: 3000}        # configs[4] is 1e5 turns (hours): the bench line times its first few thousand

# Algorithmic FP64 flops per element visit (minimal arithmetic of the
# canonical forms; FMA = 2, add/mul/sqrt/div = 1, compares = 0, sin = 1) ...
FLOPS_MIN = dict(drift=17, mult_base=2, mult_per_order=8, curved_extra=7, cavity=19, srot=12,
                 shift=2, rect=0, ellipse=5,
                 # thick maps, every operation of the canonical form counted once,
                 # sincos = 2, cosh = sinh = sqrt = division = 1, FMA = 2
                 thick_quad=66, thick_bend=68)
# ... and FP64 flops as executed by the sm_100a kernel (counted in the SASS of
# libxt_b200.so, profiles/r01_sass_fp64_counts.md): a drift is one evaluation of 1/pz and
# 1/(pz + b) (13 FP64 instructions, 21 flops; consecutive drifts share it after fusion) plus
# one application (5 instructions, 8 flops); sin and the cavity's sqrt / divisions expanded.
FLOPS_EXEC = dict(drift_eval=21, drift_apply=8, mult_base=2, mult_per_order=8, curved_extra=7, cavity=110,
                  srot=12, shift=2, rect=0, ellipse=5)


def flops_per_particle_turn(info: dict, table: dict) -> float:
    t = info["n_by_type"]
    n_mult = t[2]
    if "drift" in table:
        drifts = t[1] * table["drift"]
    else:
        drifts = info.get("n_drift_applies", t[1]) * table["drift_apply"] + info["n_drift_evals"] * table["drift_eval"]
    thick = info.get("n_thick_quad", 0) * table.get("thick_quad", 0) + info.get("n_thick_bend", 0) * table.get("thick_bend", 0)
    return (drifts + n_mult * table["mult_base"] + info["sum_order"] * table["mult_per_order"]
            + info["n_curved"] * table["curved_extra"] + t[3] * table["cavity"] + t[4] * table["srot"]
            + t[5] * table["shift"] + t[6] * table["rect"] + t[7] * table["ellipse"] + thick)


class ClockSampler:
    """Samples SM clock and throttle reasons with nvidia-smi while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


THICK_COUNTS = {}     # thick elements of the lattice make_inputs built last (xt_lattice_info counts them together)


def make_inputs(cfg: int, rank: int, workload: str = ""):
    """Seeded synthetic lattice + ensemble of config ``cfg``."""
    els = C.lattice_cfg2_thick() if workload == "thick" else C.lattice(cfg)
    buf = C.pack(els)
    THICK_COUNTS.update(n_thick_quad=sum(type(e).__name__ == "Quadrupole" for e in els),
                        n_thick_bend=sum(type(e).__name__ == "Bend" for e in els))
    if cfg in (0, 2, 3) and rank:
        coords = {0: C.particles_cfg0, 2: C.particles_cfg2, 3: C.particles_cfg3}[cfg](seed=1000 + cfg + 100 * rank)
    else:
        coords = C.particles(cfg)
    return buf, coords


def reduce_max(value: float, world: int, device) -> float:
    """MAX over ranks of a per-rank scalar (device time): the only collective of the job, outside
    every timed region.  The data path itself has none (particles are independent)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, ms_per_step: float) -> float:
    """Weak scaling: every rank tracks its own ensemble of the config's size."""
    return world * units_per_rank / (ms_per_step * 1e-3)


def oracle_sample(cfg: int, buf: bytes, coords: dict, budget_s: float = 15.0):
    """The oracle, as it stands, single-threaded, on a bounded sample of the same workload."""
    from oracle import oracle as O
    import struct
    turns_full = C.n_turns(cfg)
    n_el = struct.unpack_from("<I", buf, 12)[0]          # header field n_elements
    # calibrate on a tiny run, then size the sample for ~budget_s
    cal_n = 8
    cal = O.new_particles(buf, C.subsample(coords, slice(0, cal_n)))
    cal_turns = max(1, min(turns_full, 200000 // max(n_el, 1)))
    t0 = time.perf_counter()
    O.track(buf, cal, cal_turns)
    rate = cal_n * cal_turns * n_el / max(time.perf_counter() - t0, 1e-6)
    turns = min(turns_full, 100)
    n = int(max(8, min(len(coords["x"]), rate * budget_s / (turns * n_el))))
    p = O.new_particles(buf, C.subsample(coords, slice(0, n)))
    t0 = time.perf_counter()
    O.track(buf, p, turns)
    dt = time.perf_counter() - t0
    return {"value": n * turns * n_el / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "first %d particles of the workload x %d turns x %d elements, 1 thread, %.1f s"
                      % (n, turns, n_el, dt), "seconds": dt}


def run_reference(args):
    """--impl reference: the oracle (a deliberately plain CPU program) on the same workload,
    each step a bounded sample.  Rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    buf, coords = make_inputs(cfg, 0)
    budget = 8.0
    for _ in range(args.warmup):
        oracle_sample(cfg, buf, coords, budget_s=0.5)
    vals, secs, last = [], [], None
    for _ in range(args.steps):
        last = oracle_sample(cfg, buf, coords, budget_s=budget)
        vals.append(last["value"]); secs.append(last["seconds"])
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": WORKLOADS[cfg], "sampled": True},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": last["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def load_measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        return {}


def time_workload(X, torch, lat, coords, turns, steps, warmup, args, barrier, sampler=None):
    """W untimed + K timed steps of (restore the seeded ensemble, xt_track) on the current stream.
    -> dict(ms_per_step over the whole timed region, kernel_ms = mean CUDA-event time of the xt_track
    call alone, per-step list, alive / completed turns of the last step, launches per step)."""
    stream = torch.cuda.current_stream()
    pristine = X.new_particles(lat, coords)
    work = {k: torch.empty_like(v) for k, v in pristine.items()}

    def step(ev0=None, ev1=None):
        for k in work:
            work[k].copy_(pristine[k])
        if ev0 is not None:
            ev0.record(stream)
        X.xt_track_ex(lat, work, turns, block_size=args.block, particles_per_thread=args.ppt,
                      cold_in_registers=args.cold, balance=args.balance)
        if ev1 is not None:
            ev1.record(stream)

    for _ in range(warmup):
        step()
    barrier()
    if sampler is not None:
        sampler.start()
    launches0 = X.xt_launch_count()
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_begin.record(stream)
    for i in range(steps):
        step(*kev[i])
    t_end.record(stream)
    barrier()
    launches = X.xt_launch_count() - launches0
    clocks = sampler.stop() if sampler is not None else None
    per_step = [a.elapsed_time(b) for a, b in kev]
    out = {"total_ms": t_begin.elapsed_time(t_end), "kernel_ms": float(np.mean(per_step)),
           "kernel_ms_steps": per_step, "launches": int(launches), "clocks": clocks,
           "alive": int((work["state"] == 1).sum().item()),
           # alive particle-turns of one step (at_turn starts at 0): completed turns only
           "completed_turns": int(work["at_turn"].sum().item()),
           "work": work, "pristine": pristine}
    return out


def roofline_dict(info, n_part, turns, completed_turns, kernel_ms, peak_flops, peak_ms, n_sm, sm_max_hz):
    """FP64-ALU roofline of the tracking kernel.  `frac` counts the algorithmic
    flops of particles that were still alive (completed particle-turns); `frac_all_slots` counts every
    slot of the launch, parked lost particles included (what round 1 reported)."""
    f_min = flops_per_particle_turn(info, FLOPS_MIN)
    f_exec = flops_per_particle_turn(info, FLOPS_EXEC)
    alive_pt_per_s = completed_turns / (kernel_ms * 1e-3)
    all_pt_per_s = n_part * turns / (kernel_ms * 1e-3)
    nominal = n_sm * 64 * 2 * sm_max_hz
    return {
        "bound": "alu", "unit": "TFLOP/s",
        "achieved": f_min * alive_pt_per_s / 1e12, "peak": peak_flops / 1e12,
        "frac": f_min * alive_pt_per_s / peak_flops,
        "frac_all_slots": f_min * all_pt_per_s / peak_flops,
        # against the nominal figure from unit counts and clocks: SMs x 64 FP64 lanes x 2 x max SM clock
        "peak_nominal": nominal / 1e12, "frac_nominal": f_min * alive_pt_per_s / nominal,
        "achieved_executed": f_exec * alive_pt_per_s / 1e12, "frac_executed": f_exec * alive_pt_per_s / peak_flops,
        "peak_source": "xt_fp64_fma_peak: maximum of the DFMA microbenchmark sweep in this run (%.2f ms), burst; "
                       "nominal %d SM x 64 lanes x 2 x %.3f GHz = %.1f TFLOP/s"
                       % (peak_ms, n_sm, sm_max_hz / 1e9, nominal / 1e12),
        "kernel": "xt_track_kernel", "kernel_ms": kernel_ms,
        "flops_per_particle_turn": {"algorithmic": f_min, "executed": f_exec},
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--workload", default="", choices=["", "thick"],
                    help="thick: configs[2] with every quadrupole a thick XT_QUADRUPOLE and every bend a thick XT_BEND")
    ap.add_argument("--turns", type=int, default=0, help="override the config's turns (testing only)")
    ap.add_argument("--particles", type=int, default=0, help="override the particle count (testing only)")
    ap.add_argument("--block", type=int, default=0)
    ap.add_argument("--ppt", type=int, default=0, help="particles per thread (0: auto)")
    ap.add_argument("--chunk", type=int, default=0, help="staging-buffer bytes (0: library default)")
    ap.add_argument("--cold", type=int, default=0, help="cold state: 0 auto, 1 registers, -1 shared memory")
    ap.add_argument("--balance", type=int, default=0,
                    help="xt_track_opts.balance: 0 auto, -1 off, 1 on, n > 1 on with n turns per item")
    ap.add_argument("--also-steps", type=int, default=5, help="timed steps of the configs[2] leg (mean)")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e, cpu_baseline and configs[2] legs")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2310_00317_b200 as X

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = args.config
    turns = args.turns or BENCH_TURNS.get(cfg, C.n_turns(cfg))
    buf, coords = make_inputs(cfg, rank, args.workload)
    if args.particles:
        coords = C.subsample(coords, slice(0, args.particles))
    lat = X.xt_lattice_create_ex(buf, chunk_bytes=args.chunk) if args.chunk else X.xt_lattice_create(buf)
    info = dict(lat.info, **THICK_COUNTS)
    n_el = info["n_elements"]
    n_part = len(coords["x"])
    stream = torch.cuda.current_stream()

    # ---- roofline denominator: the maximum of the DFMA sweep, in this run
    sweep = X.xt_fp64_fma_peak_sweep()
    best = max(sweep, key=lambda r: r["tflops"])
    peak_flops, peak_ms = best["tflops"] * 1e12, best["ms"]
    props = torch.cuda.get_device_properties(local)
    n_sm = props.multi_processor_count
    peaks = load_measured_peaks()
    sm_max_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else "6650 GB/s (of fallback)"
    probe = {"dfma_three_distinct_vector_registers": X.xt_fp64_fma_probe(1)[0] / 1e12,
             "horner_4_particles_per_thread_no_lattice": X.xt_fp64_fma_probe(2)[0] / 1e12,
             "horner_same_with_uniform_register_coefficients": X.xt_fp64_fma_probe(3)[0] / 1e12}

    sampler = ClockSampler(local) if rank == 0 else None
    r = time_workload(X, torch, lat, coords, turns, args.steps, args.warmup, args, barrier, sampler)
    total_ms = reduce_max(r["total_ms"], world, "cuda")
    ms_per_step = total_ms / args.steps
    kernel_ms = r["kernel_ms"]
    units_alive = float(r["completed_turns"]) * n_el           # per rank, alive visits of one step
    units_nominal = float(n_part) * n_el * turns
    value = whole_job_value(units_alive, world, ms_per_step)
    work, pristine = r["work"], r["pristine"]

    line = None
    if rank == 0:
        wl = WORKLOADS[cfg] if not args.workload else \
            "configs[2] lattice with thick maps: 400 XT_QUADRUPOLE + 1232 XT_BEND ('expanded'), 100000 particles"
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl, "n_particles_per_gpu": n_part, "n_elements": n_el,
                       "n_turns": turns, "l2": "inputs (%.2f GB SoA per GPU) %s L2 (126 MB)" %
                                              (n_part * 13 * 8 / 1e9,
                                               "larger than" if n_part * 13 * 8 > 126e6 else "SMALLER than: the "
                                               "ensemble is re-copied from a pristine set every step and the "
                                               "kernel is ALU-bound (HBM traffic ~1e-5 of its time) against"),
                       "alive_after_step": r["alive"], "block_size": args.block or "auto",
                       "particles_per_thread": args.ppt or "auto", "records_per_turn": info["n_records"],
                       "lattice_image_bytes": info["image_bytes"], "tma_chunks_per_turn": info["n_chunks"],
                       "value_counts": "element visits of particles still alive (completed turns)"},
            "nominal_value": whole_job_value(units_nominal, world, ms_per_step),
            "particle_turns_per_s": world * n_part * turns / (ms_per_step * 1e-3),
            "alive_particle_element_turns_per_s": value,
            "gpu_launches": r["launches"],
            "clocks": r["clocks"],
            "roofline": roofline_dict(info, n_part, turns, r["completed_turns"], kernel_ms, peak_flops, peak_ms,
                                      n_sm, sm_max_hz),
        }
        line["roofline"]["kernel_ms_steps"] = r["kernel_ms_steps"]
        if cfg == 4:      # with compaction the retired slots are not tracked at all: "every slot of the launch" has no meaning
            line["roofline"]["frac_all_slots"] = None
        # DRAM bytes of one launch: not measurable inside the run (needs ncu); the number is the --set full
        # capture's dram__bytes_read + dram__bytes_write per particle scaled to this launch
        line["roofline"]["traffic"] = 45.9 * n_part * turns if cfg == 3 else None
        line["roofline"]["traffic_source"] = ("ncu capture profiles/r02i_track_cfg3_balanced_summary.md: 45.9 B per "
                                              "particle-turn (reads + writes; the state of a group of particles passes "
                                              "through HBM every four turns), scaled to the launch; not measured in "
                                              "this run") if cfg == 3 else None
        line["roofline"]["operand_pattern_ceilings_tflops"] = probe
        line["roofline"]["peak_sweep"] = {"best": best, "rows": sweep,
                                          "form": "0: fma(acc,a,b) a,b params; 1: fma(acc,x_k,b); 2: fma(acc,a,y_k)"}

    if cfg == 4 and rank == 0:
        # ---- steps C and H measured: one instrumented call (CUDA events around every pass), same workload
        for k in work:
            work[k].copy_(pristine[k])
        st = X.xt_track_ex(lat, work, turns, block_size=args.block, particles_per_thread=args.ppt, stats=True)
        ha, hb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        hist = X.xt_survival_histogram(work, 1000, 100)      # warm-up
        ha.record(stream)
        hist = X.xt_survival_histogram(work, 1000, 100)
        hb.record(stream)
        torch.cuda.synchronize()
        hist_ms = ha.elapsed_time(hb)
        gbs = st["compact_bytes"] / (st["compact_ms"] * 1e-3) / 1e9 if st["compact_ms"] > 0 else None
        passes = [{"n_in": a, "n_out": b, "ms": m, "GB/s": 2 * 112.0 * a / (m * 1e-3) / 1e9}
                  for a, b, m in zip(st["pass_n_in"], st["pass_n_out"], st["pass_ms"])]
        line["compaction"] = {
            "bound": "hbm", "unit": "GB/s", "achieved": gbs, "peak": hbm_gbs, "peak_source": hbm_src,
            "frac": gbs / hbm_gbs if gbs else None,
            "algorithmic_bytes": "2 x n_in x 112 B per pass (13 arrays + origin index read once, written once)",
            "n_passes": st["n_passes"], "compact_ms_total": st["compact_ms"], "track_ms_total": st["track_ms"],
            "share_of_call": st["compact_ms"] / (st["compact_ms"] + st["track_ms"] + st["scatter_ms"]),
            "scatter_back_ms": st["scatter_ms"],
            "scatter_back_GB/s": st["scatter_bytes"] / (st["scatter_ms"] * 1e-3) / 1e9 if st["scatter_ms"] else None,
            "passes": passes,
            "histogram": {"ms": hist_ms, "bytes": 16.0 * n_part, "GB/s": 16.0 * n_part / (hist_ms * 1e-3) / 1e9,
                          "survivors": int(hist[-1].item()), "lost_in_first_bins": [int(v) for v in hist[:4].tolist()]},
        }

    if not args.no_extras:
        # ---- e2e: the same step through xt_track_host with pinned HOST buffers (one warm-up, mean of two)
        host = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True) for k, v in pristine.items()}
        host0 = {k: v.cpu() for k, v in pristine.items()}
        e2e_runs = []
        for it in range(3):
            for k in host:
                host[k].copy_(host0[k])
            barrier()
            t0 = time.perf_counter()
            X.xt_track_host(lat, host, turns, block_size=args.block, particles_per_thread=args.ppt)  # synchronises itself
            barrier()
            if it:
                e2e_runs.append(time.perf_counter() - t0)
        e2e_s = float(np.mean(e2e_runs))
        e2e_max = reduce_max(e2e_s, world, "cuda")
        if rank == 0:
            nbytes = sum(v.numel() * 8 for v in host.values())
            done = float(host["at_turn"].sum().item())
            line["e2e"] = {"value": world * done * n_el / e2e_max, "unit": UNIT,
                           "nominal_value": world * units_nominal / e2e_max,
                           "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                           "seconds": e2e_max, "runs": e2e_runs, "api": "xt_track_host (pinned host SoA)",
                           "alive_after_step": int((host["state"] == 1).sum().item())}
        del host, host0
    del work, pristine, r
    lat.close()
    torch.cuda.empty_cache()

    if rank == 0 and not args.no_extras:
        # ---- configs[2] (the other configuration the north_star's target names), same run, same peak:
        #      mean over >= 5 timed steps after 3 warm-up steps, with its own roofline
        if cfg == 3 and world == 1:
            b2, c2 = make_inputs(2, 0)
            l2 = X.xt_lattice_create(b2)
            assert not THICK_COUNTS["n_thick_quad"]
            t2 = C.n_turns(2)
            n2 = len(c2["x"])
            r2 = time_workload(X, torch, l2, c2, t2, max(5, args.also_steps), 3, args, barrier)
            ms2 = r2["total_ms"] / max(5, args.also_steps)
            line["also"] = {"workload": WORKLOADS[2], "value": r2["completed_turns"] * l2.info["n_elements"] / (ms2 * 1e-3),
                            "nominal_value": float(n2) * t2 * l2.info["n_elements"] / (ms2 * 1e-3),
                            "unit": UNIT, "steps": max(5, args.also_steps), "warmup": 3, "ms_per_step": ms2,
                            "alive_after_step": r2["alive"],
                            "roofline": roofline_dict(l2.info, n2, t2, r2["completed_turns"], r2["kernel_ms"],
                                                      peak_flops, peak_ms, n_sm, sm_max_hz)}
            line["also"]["roofline"]["kernel_ms_steps"] = r2["kernel_ms_steps"]
            line["also"]["frac"] = line["also"]["roofline"]["frac"]
            del r2
            l2.close()
        # ---- cpu_baseline: the oracle as it stands on a bounded sample of the same workload
        line["cpu_baseline"] = {k: v for k, v in oracle_sample(cfg, buf, coords).items() if k != "seconds"}
        line["cpu_baseline"]["host_cores_on_this_box"] = os.cpu_count()
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
