#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the B200 beam-tracking hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload fodo_channel|...]

Metric (BASELINE.json): particle-element pushes/s (fp64).  One *element push* = one particle through one
lattice element (all its slices).  Workload at N=1 = BASELINE configs[1] ("Linear FODO channel": 10^6
particles, the FODO cell x100 = 500 elements / 5300 slice maps, 1 pass), synthetic seeded input from
workloads/.  A *step* = one pass of the hot path over the bunch = one bt_track(1) call = ONE kernel launch.

N > 1 (torchrun): particles are independent, so the path shards with no data-path collective; every rank
tracks its own 10^6-particle bunch (seed + rank) -> "scaling": "weak"; value = all ranks' pushes / max-over-ranks time.

Timing: W >= 3 warm-up steps; every timed step is bracketed by CUDA events on the beam's stream (torch's current
stream); L2 is flushed (256 MiB write) between timed steps, outside the event intervals; the K-step region is
bracketed by barrier + torch.cuda.synchronize(); ms_per_step = sum of event intervals / K, max over ranks.

The same JSON line carries: roofline (FP64-pipe issue slots), cpu_baseline (the oracle as
it stands on a bounded sample, host cores), e2e (host pinned buffers -> bt_track_host = chunked upload -> bt_track ->
bt_beam_download inside the timed region), gpu_launches, clocks.
"""
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
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "particle-element pushes/s (fp64)"
UNIT = "pushes/s"

# FP64 issue slots per slice map (DESIGN.md section 7 / SURVEY 8d): minimal DFMA/DMUL sequences.
SLOTS = {"drift": 3, "quad": 9, "sbend": 10, "dipedge": 2, "shortrf": 4}


def slots_per_particle_per_turn(lattice):
    total = 0
    for el in lattice:
        kind, ns = el[0], el[2]
        if kind == "multipole":
            m, ks = int(el[3]), el[5]
            per = 5 if (m == 3 and ks == 0.0) else 8 if (m == 4 and ks == 0.0) else 4 * max(m - 1, 0) + 6
        elif kind == "quad" and el[3] == 0.0:
            per = SLOTS["drift"]
        else:
            per = SLOTS[kind]
        total += per * ns
    return total


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.QUERY,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])), mx.append(float(f[1])), pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def get_workload(name, rank):
    idx = {"tiny_fodo": 0, "fodo_channel": 1, "chicane": 2, "nonlinear_ring": 3}[name]
    cfg = W.config(idx)
    from paper_2208_02382_b200.shard import rank_seed
    cfg.seed = rank_seed(cfg.seed, rank)   # every rank its own bunch (weak scaling)
    return cfg


# ---------------------------------------------------------------------------------------------------
# reference arm: the oracle as it stands, on the host cores, on a bounded sample of the same workload
# ---------------------------------------------------------------------------------------------------
def oracle_rate(cfg, n_sample, reps=1):
    import oracle as O
    coords = W.make_bunch(cfg, n=n_sample)
    g0 = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    times = []
    for _ in range(reps):
        c = [a.copy() for a in coords]
        t0 = time.perf_counter()
        O.track(c, cfg.lattice, cfg.nturns, g0)
        times.append(time.perf_counter() - t0)
    pushes = n_sample * cfg.n_elements * cfg.nturns
    return pushes, times, O.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = get_workload(args.workload, 0)
    # W warm-up steps on a small sample also calibrate the rate; the per-step sample is then sized so that the
    # K timed steps take about REF_BUDGET_S seconds in total (bounded sample of the same workload).
    REF_BUDGET_S = 60.0
    n_cal = min(cfg.n, 20_000)
    rate = None
    for _ in range(max(1, args.warmup)):
        p, tms, _c = oracle_rate(cfg, n_cal)
        rate = n_cal / tms[0]                                   # particles (through the full lattice) per second
    n_sample = args.ref_sample if args.ref_sample > 0 else int(rate * REF_BUDGET_S / max(1, args.steps))
    n_sample = max(1000, min(cfg.n, n_sample))
    pushes, times, cores = oracle_rate(cfg, n_sample, reps=max(1, args.steps))
    t = sum(times) / len(times)
    value = pushes / t
    sample = "%d of %d particles (seed %d), full lattice (%d elements, %d slice maps), %d turn(s) per step" % (
        n_sample, cfg.n, cfg.seed, cfg.n_elements, cfg.slice_maps_per_turn, cfg.nturns)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": len(times),
        "warmup": max(1, args.warmup), "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[1] " + cfg.name + " (bounded sample)", "particles": n_sample,
                   "elements": cfg.n_elements, "slice_maps_per_turn": cfg.slice_maps_per_turn, "turns": cfg.nturns},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------
# the rest of the hot path (N = 1): the other tracking configs and the space-charge kernels of configs[4]
# ---------------------------------------------------------------------------------------------------
def _event_ms(torch, fn, reps, flush, pre=None):
    """CUDA-event time of fn() on the current stream; L2 flushed (and `pre` run) before each repetition, outside."""
    ts = []
    for _ in range(reps):
        if pre:
            pre()
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return ts


def bench_other_configs(bt, torch, flush, peaks, nominal_peak):
    """bt_track on configs[0], [2], [3] at full size (one call = the config's nturns).  configs[3]'s 64e6-particle
    bunch is a seeded 10^6-particle draw tiled 64 times on the device (timing does not depend on the values)."""
    out = []
    hbm = float(peaks["hbm_gbs"]) * 1e9
    for idx, reps in ((0, 5), (2, 5), (3, 2)):
        cfg = W.config(idx)
        n = cfg.n
        base = W.make_bunch(cfg, n=min(n, 1_000_000))
        tile = -(-n // len(base[0]))
        pristine = [torch.from_numpy(a).cuda().repeat(tile)[:n].contiguous() for a in base]
        beam = bt.Beam(n)
        beam.lattice_set(cfg.lattice)

        def restore():
            for d, s in zip(beam.tensors, pristine):
                d.copy_(s)
            beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)   # RF lattices: same energy every repetition

        restore()
        beam.track(cfg.nturns)
        launches0 = bt.launch_count()
        ts = _event_ms(torch, lambda: beam.track(cfg.nturns), reps, flush, restore)
        launches = (bt.launch_count() - launches0) // reps
        t = statistics.mean(ts) * 1e-3
        slots = float(n) * slots_per_particle_per_turn(cfg.lattice) * cfg.nturns
        t_alu, t_hbm = slots / nominal_peak, 96.0 * n * launches / hbm
        li = beam.last_launch()
        entry = {"workload": "configs[%d] %s" % (idx, cfg.name), "particles": n, "elements": cfg.n_elements, "turns": cfg.nturns,
                 "ms_per_call": t * 1e3, "pushes_per_s": n * cfg.n_elements * cfg.nturns / t, "launches_per_call": launches,
                 "kernel": "bt::track_kernel<P=%d> grid=%d block=%d" % (li["particles_per_thread"], li["grid"], li["block"])}
        if idx == 0:
            entry["roofline"] = {"bound": "latency", "note": "10^4 particles = 313 warps on 148 SMs: neither pipe nor HBM can be filled "
                                 "(SURVEY 8d); roofline time %.2f us shown for information" % (max(t_alu, t_hbm) * 1e6)}
        elif t_alu >= t_hbm:
            entry["roofline"] = {"bound": "alu", "achieved": slots / t / 1e12, "peak": nominal_peak / 1e12, "unit": "Tslot/s",
                                 "frac": t_alu / t}
        else:
            entry["roofline"] = {"bound": "hbm", "achieved": 96.0 * n * launches / t / 1e9, "peak": hbm / 1e9, "unit": "GB/s",
                                 "frac": t_hbm / t}
        if idx in (2, 3):
            # beam statistics: bt_beam_moments = 1 launch + a 336-byte read-back, 48 B/particle
            beam.moments()
            tm = statistics.mean(_event_ms(torch, beam.moments, 5, flush)) * 1e-3
            entry["moments"] = {"ms": tm * 1e3, "roofline": {"bound": "hbm", "achieved": 48.0 * n / tm / 1e9, "peak": hbm / 1e9,
                                                              "unit": "GB/s", "frac": 48.0 * n / tm / hbm, "traffic": None}}
        out.append(entry)
        beam.close()
        del pristine, beam
        torch.cuda.empty_cache()
    return out


def bench_spacecharge(bt, torch, flush, peaks):
    """configs[4] A and B at full size (8e6 particles, 128^3 nodes): bt_beam_sort_by_cell once, then 10 steps of
    bt_deposit_cic + bt_gather_kick(0, ds) (SURVEY 8d call sequence), every call timed with CUDA events, L2 flushed
    before each.  GB/s = ALGORITHMIC bytes / time: deposit 24 B/particle + 2 x 8 B/node (zeroing + result);
    gather+kick+drift 96 B/particle + 24 B/node."""
    hbm = float(peaks["hbm_gbs"])
    out = {}
    for variant, order in (("A", 1), ("B", 1), ("A", 2)):
        sc = W.spacecharge_config(variant)
        c = W.make_spacecharge_bunch(sc)
        E = W.gaussian_bunch_field(sc)
        n, nn = sc.n, sc.shape[0] * sc.shape[1] * sc.shape[2]
        dep_bytes, gat_bytes = 24.0 * n + 16.0 * nn, 96.0 * n + 24.0 * nn
        beam, grid = bt.Beam(n), bt.Grid(sc.shape, sc.lo, sc.d)
        beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
        grid.set_particle_shape(order)                             # 1 = CIC (configs[4]); 2 = the listing's shape (S:8f NEXT-2)
        grid.set_field(*E)
        beam.lattice_set([("drift", sc.ds / 2, 1)])
        beam.upload(c)
        beam.track(1)                                              # leading half drift
        # unsorted (caller's order), one call each, for information
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)       # warm-up
        t_dep_u = min(_event_ms(torch, lambda: beam.deposit_cic(grid, sc.q_weight, sc.zscale, True), 2, flush))
        pos = [t.clone() for t in beam.tensors]
        t_gat_u = min(_event_ms(torch, lambda: beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, 0.0), 2, flush))
        for d, s in zip(beam.tensors, pos):
            d.copy_(s)
        del pos
        beam.sort_by_cell(grid, sc.zscale)                         # warm-up: first call allocates the scratch
        beam.upload(c)                                             # back to the caller's order
        beam.track(1)
        t_sort = _event_ms(torch, lambda: beam.sort_by_cell(grid, sc.zscale), 1, flush)[0]
        t_dep, t_gat = [], []
        for step in range(sc.nsteps):
            t_dep += _event_ms(torch, lambda: beam.deposit_cic(grid, sc.q_weight, sc.zscale, True), 1, flush)
            after = sc.ds if step < sc.nsteps - 1 else sc.ds / 2
            t_gat += _event_ms(torch, lambda: beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, after), 1, flush)
        poisson = None
        if variant == "A" and order == 1:
            # NEXT-4: rest-frame Poisson solve on the deposited rho (own kernels + 2 cuFFT transforms of the 256^3 padded
            # box); the prescribed field is put back afterwards.  Bytes = one read and one write per array per pass if
            # each FFT were a single pass over its data (a lower bound on HBM traffic): 1.0 GB at 128^3
            # (padded box = 8 nn reals, spectrum = 4 nn complex, real Green transform = 4 nn reals).
            gz = 1.0 + sc.kin_energy_MeV / sc.mass_MeV
            grid.solve_poisson(gz)                                 # warm-up: plans, buffers, Green transform
            t_ps = _event_ms(torch, lambda: grid.solve_poisson(gz), 5, flush)
            ps_bytes = 8.0 * nn * ((1 + 1) + (8 + 8) + (8 + 4 + 8) + (8 + 8) + (1 + 1 + 4))   # in doubles per node: copy, D2Z, multiply, Z2D, gradient
            mp_ = statistics.mean(t_ps) * 1e-3
            poisson = {"ms": mp_ * 1e3, "padded_box": [2 * s for s in sc.shape],
                       "roofline": {"bound": "hbm", "achieved": ps_bytes / mp_ / 1e9, "peak": hbm, "unit": "GB/s",
                                    "frac": ps_bytes / mp_ / 1e9 / hbm, "traffic": None,
                                    "note": "bytes = single-pass lower bound of the pad/FFT/multiply/FFT/extract/gradient chain"}}
            grid.set_field(*E)
        md, mg = statistics.mean(t_dep) * 1e-3, statistics.mean(t_gat) * 1e-3
        out[variant if order == 1 else variant + "_order2"] = {
            "workload": "configs[4] %s, %d particles, %dx%dx%d nodes, %d steps, particle shape order %d" % (
                (sc.name, n) + tuple(sc.shape) + (sc.nsteps, order)),
            "sort_by_cell_ms_once": t_sort,
            "deposit": {"ms": md * 1e3, "ms_first_last": [t_dep[0], t_dep[-1]], "unsorted_ms": t_dep_u,
                        "roofline": {"bound": "hbm", "achieved": dep_bytes / md / 1e9, "peak": hbm, "unit": "GB/s",
                                     "frac": dep_bytes / md / 1e9 / hbm, "traffic": None}},
            "gather_kick_drift": {"ms": mg * 1e3, "ms_first_last": [t_gat[0], t_gat[-1]], "unsorted_kick_only_ms": t_gat_u,
                                  "roofline": {"bound": "hbm", "achieved": gat_bytes / mg / 1e9, "peak": hbm, "unit": "GB/s",
                                               "frac": gat_bytes / mg / 1e9 / hbm, "traffic": None}},
            "ms_per_step_incl_sort_amortised": (md + mg) * 1e3 + t_sort / sc.nsteps,
        }
        if poisson:
            out[variant]["poisson_solve"] = poisson
        beam.close()
        grid.close()
        del beam, grid
        torch.cuda.empty_cache()
    return out


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2208_02382_b200 as bt

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = get_workload(args.workload, rank)
    coords = W.make_bunch(cfg)
    n = cfg.n
    pushes_per_step = n * cfg.n_elements * cfg.nturns
    slots_pp = slots_per_particle_per_turn(cfg.lattice) * cfg.nturns
    slots_per_launch = float(n) * slots_pp

    beam = bt.Beam(n)                       # six torch.float64 CUDA tensors lent to the library
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(cfg.lattice)
    pinned = [torch.from_numpy(a).pin_memory() for a in coords]
    pinned_out = [torch.empty(n, dtype=torch.float64).pin_memory() for _ in range(6)]
    pristine = [t.to("cuda", non_blocking=True) for t in pinned]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def restore():
        for dst, src in zip(beam.tensors, pristine):
            dst.copy_(src, non_blocking=True)

    # ---- device-resident timing ----------------------------------------------------------------
    restore()
    for _ in range(max(args.warmup, 3)):
        beam.track(cfg.nturns)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = bt.launch_count()
    barrier()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        restore()                            # same input every step (outside the event interval)
        flush.zero_()                        # L2 flush between timed iterations (outside the event interval)
        ev[k][0].record()
        beam.track(cfg.nturns)               # ONE fused-walk launch
        ev[k][1].record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = bt.launch_count() - launches0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    ms_sum = sum(step_ms)

    launch_info = beam.last_launch()         # geometry of the timed launches (the e2e leg below launches per chunk)

    # ---- end to end through the C-ABI with host buffers -----------------------------------------
    # bt_track_host = upload + walk + download with the bunch cut into chunks on three streams (copies overlap the walk)
    for _ in range(2):
        beam.track_host(pinned, pinned_out, cfg.nturns, args.e2e_chunks)
    barrier()
    t0 = time.perf_counter()
    for k in range(args.steps):
        beam.track_host(pinned, pinned_out, cfg.nturns, args.e2e_chunks)     # synchronous: returns when pinned_out is complete
    barrier()
    t_e2e = time.perf_counter() - t0
    clocks = sampler.stop() if rank == 0 else None

    # max over ranks
    from paper_2208_02382_b200.shard import max_over_ranks
    ms_sum, t_e2e, t_wall = max_over_ranks([ms_sum, t_e2e, t_wall], device="cuda")

    result = None
    if rank == 0:
        peaks, peaks_kind = load_peaks()
        ms_per_step = ms_sum / args.steps
        value = world * pushes_per_step / (ms_per_step * 1e-3)
        e2e_value = world * pushes_per_step * args.steps / t_e2e
        # roofline of the dominant (only) kernel: FP64 pipe issue slots
        nominal_peak = 148 * 64 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6       # slots/s at max SM clock
        measured_fp64 = bt.calib_fp64(300.0)
        measured_rw6 = bt.calib_rw6(min(64_000_000, max(n, 8_000_000)), 5)
        achieved = slots_per_launch / (statistics.mean(step_ms) * 1e-3)
        hbm_time_ms = 96.0 * n / (float(peaks["hbm_gbs"]) * 1e9) * 1e3
        alu_time_ms = slots_per_launch / nominal_peak * 1e3
        bound = "alu" if alu_time_ms >= hbm_time_ms else "hbm"
        if bound == "alu":
            roof = {"bound": "alu", "achieved": achieved / 1e12, "peak": nominal_peak / 1e12, "unit": "Tslot/s",
                    "frac": achieved / nominal_peak,
                    # dram__bytes_read.sum + dram__bytes_write.sum of one launch on configs[1] from the ncu --set full capture in
                    # profiles/r01_summary.md (48.0 MB read + 1.1 MB written: the 48 MB result stays in the 126 MB L2);
                    # algorithmic bytes 96 B/particle = 96 MB per launch.  null for any other workload (not captured).
                    "traffic": 49.1e6 if (args.workload == "fodo_channel" and n == 1_000_000) else None,
                    "traffic_unit": "bytes per launch (ncu, profiles/r01_summary.md)",
                    "peak_kind": "derived: 148 SMs x 64 FP64 lanes x %s sm_max_mhz (DESIGN.md s7)" % peaks_kind,
                    "peak_measured_dfma_chain": measured_fp64 / 1e12, "frac_of_measured_dfma_chain": achieved / measured_fp64,
                    "slots_per_particle": slots_pp, "tflops": None}
        else:
            gbs = 96.0 * n / (statistics.mean(step_ms) * 1e-3) / 1e9
            roof = {"bound": "hbm", "achieved": gbs, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
                    "frac": gbs / float(peaks["hbm_gbs"]), "traffic": None, "peak_kind": peaks_kind + " copy bandwidth",
                    "rw6_stream_ceiling_gbs": measured_rw6}
        roof["kernel"] = "bt::track_kernel<P=%d> grid=%d block=%d smem=%dB" % (
            launch_info["particles_per_thread"], launch_info["grid"], launch_info["block"], launch_info["smem_bytes"])
        roof["roofline_time_ms"] = max(alu_time_ms, hbm_time_ms)
        roof["rw6_stream_ceiling_gbs"] = measured_rw6
        # CPU baseline: the oracle as it stands, bounded sample, host cores
        cb_cfg = get_workload(args.workload, 0)
        n_cb = min(n, 1_000_000)
        cb_times, cores, cb_pushes = [], 0, 0
        while sum(cb_times) < 10.0 and len(cb_times) < 12:       # about 10-30 s of CPU work
            cb_pushes, tms, cores = oracle_rate(cb_cfg, n_cb)
            cb_times += tms
        cb_t = sum(cb_times) / len(cb_times)
        cpu_baseline = {"value": cb_pushes / cb_t, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": "%d of %d particles, full lattice (%d slice maps), %d turn(s); %d repetitions, %.1f s of CPU work in total"
                                  % (n_cb, n, cfg.slice_maps_per_turn, cfg.nturns, len(cb_times), sum(cb_times))}
        # the same oracle on ONE thread (SURVEY 8d asks for both), on a smaller sample of the same workload (~3 s)
        try:
            import oracle as _O
            nthr = _O.num_threads()
            _O.set_num_threads(1)
            n_st = min(n_cb, 100_000)
            st_pushes, st_times, _ = oracle_rate(cb_cfg, n_st)
            _O.set_num_threads(nthr)
            cpu_baseline["single_thread"] = {"value": st_pushes / st_times[0], "unit": UNIT, "cores": 1,
                                             "sample": "%d of %d particles, full lattice, %d turn(s), one run" % (n_st, n, cfg.nturns)}
        except Exception as exc:  # the all-cores number above is the contract; this one is extra
            cpu_baseline["single_thread"] = {"unavailable": repr(exc)}
        extras = {}
        if world == 1 and not args.no_extras:
            extras["other_configs"] = bench_other_configs(bt, torch, flush, peaks, nominal_peak)
            extras["spacecharge"] = bench_spacecharge(bt, torch, flush, peaks)
        result = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[1] " + cfg.name, "particles_per_gpu": n, "elements": cfg.n_elements,
                       "slice_maps_per_turn": cfg.slice_maps_per_turn, "turns_per_step": cfg.nturns,
                       "slice_maps_per_s": world * n * cfg.slice_maps_per_turn * cfg.nturns / (ms_per_step * 1e-3),
                       "l2": "flushed between timed steps (256 MiB write)", "parallelism": "particles sharded, %d rank(s), no collective" % world},
            "roofline": roof, "cpu_baseline": cpu_baseline,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 48 * n, "d2h_bytes_per_step": 48 * n,
                    "ms_per_step": t_e2e / args.steps * 1e3,
                    "call": "bt_track_host(pinned in, pinned out, nturns, nchunks=%d): H2D / walk / D2H of the chunks overlap "
                            "on three streams" % args.e2e_chunks},
            "gpu_launches": int(launches), "clocks": clocks,
            "step_ms_min_median_max": [min(step_ms), statistics.median(step_ms), max(step_ms)],
            "wall_s_timed_region": t_wall,
        }
        result.update(extras)
    beam.close()
    if world > 1:
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(result), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="fodo_channel", choices=["tiny_fodo", "fodo_channel", "chicane", "nonlinear_ring"])
    ap.add_argument("--ref-sample", type=int, default=0,
                    help="particles per step the oracle is timed on in --impl reference (0 = sized for ~60 s in total)")
    ap.add_argument("--e2e-chunks", type=int, default=8, help="chunks of the bunch in bt_track_host (e2e leg)")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the other configs and the space-charge kernels (N=1 only; the headline is unchanged)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
