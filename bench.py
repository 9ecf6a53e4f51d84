#!/usr/bin/env python
"""bench.py -- throughput of the symplectic lattice step (arXiv 1201.5029 §2.3) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4_chaotic512] [--order 4]
                    [--precision 64] [--impl ours|reference]
    python bench.py --sweep cfg4      # BASELINE.json configs[4]: 512^3, 1024^3 x fp64, fp32 x order 2, 4, 6, 50 steps
                                      # each, one JSON line per cell (device-generated initial conditions)

One "step" is one whole composite step of the chosen order (all stages: merged drift + kick + lattice sums +
scalar update) over the whole lattice.  The metric is BASELINE.json's: lattice
site-updates per second per field, SU/s = N^3 * nfields * steps / time.  One JSON line on stdout (rank 0).

  value     inputs resident in HBM; CUDA events on the launching stream around K steps (one pycool_step(K)).
  e2e       same job from pinned HOST buffers to HOST buffers through the public API: set_fields (H2D), K steps,
            energies, read_fields (D2H), all inside the timed region.
  roofline  the fused drift+kick kernel: algorithmic bytes per launch (4 * sizeof(real) per field-site)
            / its average duration, bracketed per launch by CUDA events in a second pass of the same K steps
            (brackets between launches would switch off the launch overlap the first, timed pass runs with).
            bound / traffic come from the committed ncu --set full summary of the SAME launch geometry
            (profiles/kick_counters.txt, keyed by workload, precision, kernel variant and z-chunk); when the live
            geometry has no capture they are reported as unknown, never carried over from another geometry.
  cpu_baseline  the CPU oracle, as it stands, on a bounded sub-lattice of the same workload (1 thread): an accuracy
            reference (three passes per stage, compensated long-double sums), NOT a tuned CPU implementation.
--impl reference times that oracle alone (there is no reference implementation to install: the paper ships no
code).  Multi-GPU: the path does not shard (north_star: one GPU); --gpus N runs N
independent replicas, one per rank ("replicas only", weak scaling, no collective on the data path).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "lattice site-updates/sec (fp64, per field)"
UNIT = "site-updates/s"
ORACLE_SAMPLE_N = 64          # sub-lattice the oracle is timed on (same dx, dt, model, order)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4_chaotic512")
    ap.add_argument("--order", type=int, default=None)
    ap.add_argument("--precision", type=int, default=64, choices=[32, 64])
    ap.add_argument("--tile", type=int, default=-1)
    ap.add_argument("--zchunk", type=int, default=0)
    ap.add_argument("--item-order", type=int, default=-1, help="tiles per region of the item order (0: plain x-y-z; -1: library's)")
    ap.add_argument("--persistent", type=int, default=-1, help="1/0: persistent launch of the TMA kernel on/off (default: library's)")
    ap.add_argument("--cooperative", type=int, default=-1, help="1/0: multi-stage cooperative launches on small lattices on/off (default: library's)")
    ap.add_argument("--fused-tail", type=int, default=-1, help="1/0: fused stage tail on/off (default: library's)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-init", action="store_true", help="skip the on-device initial-conditions timing")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-linear", action="store_true", help="skip the linearised-solver block (SURVEY 8(f) rank 4)")
    ap.add_argument("--device-init", action="store_true",
                    help="initial conditions from pycool_init_fields instead of host arrays (no e2e): for 1024^3 captures")
    ap.add_argument("--sweep", default=None, choices=["cfg4"], help="print the configs[4] matrix, one JSON line per cell")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


COUNTER_COLUMNS = ("dram_bytes", "duration_us", "dram_pct", "fp64_pct", "issue_pct", "warps_active_pct", "l2_hit_pct")


def geometry_key(workload, precision, geo):
    return "%s/fp%d/tile%d/zc%d/region%dx%d" % ((workload, precision, geo["variant"], geo["zchunk"]) + tuple(geo["region"]))


def recorded_counters(key):
    """Per-launch ncu --set full counters of the fused kernel for exactly this workload, precision, kernel variant and
    z-chunk, from the committed summary profiles/kick_counters.txt (lines "<key> <dram bytes> <duration us>
    <dram %> <fp64 pipe %> <issue slots %> <warps active %> <L2 hit %>"), or None when that geometry has no capture."""
    p = os.path.join(ROOT, "profiles", "kick_counters.txt")
    try:
        for line in open(p):
            w = line.split()
            if len(w) == 1 + len(COUNTER_COLUMNS) and w[0] == key:
                return dict(zip(COUNTER_COLUMNS, (float(x) for x in w[1:])))
    except OSError:
        pass
    return None


def bound_from_counters(c):
    """What the counters of the capture say limits the kernel: "hbm" when DRAM throughput is the busiest unit and it
    is busy (>= 70 % of its peak); "alu" when the fp64 pipe or the issue slots are; otherwise the kernel waits on
    latency with every unit partly idle -- then the roofline it is measured against stays HBM (the unit it would
    saturate first: the busiest one) and `limiter` says so."""
    units = {"dram": c["dram_pct"], "fp64 pipe": c["fp64_pct"], "issue slots": c["issue_pct"]}
    top = max(units, key=units.get)
    desc = ", ".join("%s %.0f %%" % kv for kv in units.items()) + ", warps active %.0f %%" % c["warps_active_pct"]
    if units[top] < 70.0:
        return "hbm", "latency/occupancy: no unit above 70 %% busy (%s); busiest: %s" % (desc, top)
    return ("hbm" if top == "dram" else "alu"), "%s (%s)" % (top, desc)


def host_description():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def wait_first(self, timeout=3.0):
        """Block until nvidia-smi has delivered its first line (it needs ~0.1-1 s to start), so that samples fall
        inside the warm-up and the timed region even when those last only tens of milliseconds."""
        t0 = time.time()
        while self.proc and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.01)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        busy = [x for x in sm if mx and x > 0.5 * mx] or sm
        med = busy[len(busy) // 2] if busy else None
        return {"sm_mhz": med, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(x, world, device):
    """MAX over ranks of one host float (the slowest rank's time); identity at world 1.  Needs an initialised
    process group (NCCL on GPUs; the CPU tests drive it over gloo)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(N, nf, steps, world, seconds):
    """Replicas only: every rank steps its own lattice, so the job's units are world x one rank's,
    over the slowest rank's time."""
    return float(N) ** 3 * nf * steps * world / seconds


def time_oracle(cfg, order, steps, warmup, precision):
    """The oracle on an ORACLE_SAMPLE_N^3 sub-lattice with the workload's dx, dt, model and order."""
    import oracle
    from paper_1201_5029_b200 import inputs
    n = min(ORACLE_SAMPLE_N, cfg["N"])
    sub = dict(cfg)
    sub["N"], sub["L"] = n, cfg["L"] * n / cfg["N"]
    phi, pi = inputs.make_initial(sub, precision=precision, fft_max=n)
    o = oracle.Oracle(n, sub["L"], sub["nfields"], sub["model"], sub["p"], order=order, dt=cfg["dt"],
                      mpl=sub["mpl"], rho_gamma0=sub["rho_gamma0"], rho_m0=sub["rho_m0"], precision=precision)
    o.set_fields(phi, pi)
    o.set_background(1.0)
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    units = float(n) ** 3 * sub["nfields"] * steps
    sample = "%d^3 sub-lattice of %s (same dx, dt, model, order %d), %d steps, %.1f s" % (n, cfg["name"], order, steps, dt)
    return units / dt, dt / steps * 1e3, sample


ORACLE_NOTE = ("accuracy oracle: three passes per stage, Neumaier-compensated long-double sums, -ffp-contract=off, "
               "1 thread; not a tuned CPU implementation and not a speed-up denominator")


def cpu_baseline_block(v, sample):
    d = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "note": ORACLE_NOTE}
    d.update(host_description())
    return d


def timed_steps(lat, steps, barrier, stream):
    """EXACTLY `steps` steps (one pycool_step call + the deferred closing drift) between two CUDA events on the
    context's stream, nothing else in the stream.  Returns milliseconds."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    lat.step(steps)
    lat.flush()                  # the deferred closing half drift belongs to these steps: inside the timed region
    e1.record(stream)
    barrier()
    return e0.elapsed_time(e1)


def roofline_block(lat, workload, precision, N, nf, steps, barrier):
    """Second pass of the same `steps` steps with every fused drift+kick launch bracketed by CUDA events on the same
    stream (pycool_set_profiling); the whole pass is timed too, for the kernel's share of a step."""
    lat.sync()
    time.sleep(1.0)              # let the board's power average recover, so both passes start from the same state
    lat.step(1)                  # (untimed) clocks back up
    lat.set_profiling(True)
    ms_prof = timed_steps(lat, steps, barrier, lat.stream)
    kick_ms, kick_n = lat.kick_time_ms()
    lat.set_profiling(False)
    peak, peak_src = measured_peaks()
    esz = precision // 8
    alg_bytes = 4.0 * esz * N ** 3 * nf                       # read phi, pi; write phi, pi
    kick_avg_ms = kick_ms / max(kick_n, 1)
    achieved = alg_bytes / (kick_avg_ms * 1e-3) / 1e9
    geo = lat.kick_geometry()
    key = geometry_key(workload, precision, geo)
    cnt = recorded_counters(key)
    roof = {"bound": "hbm", "kernel": "kick_tma" if geo["tma_stages"] > 0 else "kick_fused", "achieved": achieved,
            "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src, "traffic": None,
            "algorithmic_bytes_per_launch": alg_bytes, "launches_timed": kick_n, "avg_launch_ms": kick_avg_ms,
            "kernel_share_of_step": kick_ms / ms_prof, "geometry": geo, "capture_key": key,
            # both denominators -- the measured copy peak above and B200's nominal 8 TB/s
            "nominal_peak": 8000.0, "frac_of_nominal": achieved / 8000.0,
            "measured": "second pass of the same %d steps with every launch bracketed by CUDA events" % steps}
    if cnt:
        roof["bound"], roof["limiter"] = bound_from_counters(cnt)
        roof["traffic"] = cnt["dram_bytes"]
        roof["traffic_over_algorithmic"] = cnt["dram_bytes"] / alg_bytes
        roof["ncu"] = cnt
        roof["bound_source"] = "ncu --set full capture of this geometry (profiles/kick_counters.txt)"
    else:
        roof["bound_source"] = ("assumed: no committed ncu capture for %s (traffic unknown, never carried over from "
                                "another geometry)" % key)
    return roof


def linear_block(dev, N=256, steps=20):
    """SURVEY 8(f) rank 4, on demand: the linearised solver (include/pycool_linear.h) on the two-field chaotic model,
    N^3 modes, order 4: `steps` steps through the growth matrices (2.51) against the same steps with every mode on
    its own -- the comparison behind the paper's "roughly 15 times faster".  Device times of the
    kernels from CUDA events inside the library; second of two identical calls."""
    import numpy as np
    from paper_1201_5029_b200 import binding
    peak, _ = measured_peaks()
    out = {"workload": "chaotic model, %d^3, 2 fields, order 4, %d steps per call" % (N, steps)}
    rng = np.random.default_rng(11)
    shape = (2, N, N, N // 2 + 1)
    P = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * 1e-6
    for name, method in (("growth", binding.GROWTH), ("naive", binding.NAIVE)):
        g = binding.LinearLattice(N, 10.0, 2, binding.CHAOTIC, (1.0, 1.0e4), order=4, dt=10.0 / N / 20.0, device=dev)
        g.set_background(1.0, float("nan"), (0.9676, 0.0), (-0.71371, 0.0))
        g.set_modes(P, P)
        g.step(steps, method)
        g.step(steps, method)
        t = g.time_ms()
        t["total"] = t["background"] + t["growth"] + t["modes"]
        out[name + "_ms"] = t
        if method == binding.GROWTH:
            nmodes, ncls = N * N * (N // 2 + 1), g.nclasses
            # lin_apply: 2 nf complex read + written per mode, one (2 nf)^2 matrix read per class (the gathers of the
            # ~23 modes of a class hit L2)
            alg = nmodes * 4 * 16 * 2 + ncls * 16 * 8
            out["apply"] = {"algorithmic_bytes": alg, "achieved": alg / (t["modes"] * 1e-3) / 1e9, "unit": "GB/s",
                            "frac": alg / (t["modes"] * 1e-3) / 1e9 / peak, "bound": "hbm"}
            # lin_growth: per class, column and stage 2 nf + nf (1 + nf) = 10 fp64 FMAs (nf = 2)
            fma = ncls * 4 * steps * 3 * 10
            out["growth_kernel"] = {"fp64_fma": fma, "achieved": 2 * fma / (t["growth"] * 1e-3) / 1e12, "unit": "TFLOP/s",
                                    "bound": "alu"}
            out["classes"], out["modes"] = ncls, nmodes
        g.close()
    out["speedup_growth_over_naive"] = out["naive_ms"]["total"] / out["growth_ms"]["total"]
    out["paper"] = "roughly 15 times faster than the naive version (PAPER.md:403, Fermi-class GPU)"
    return out


def sweep_cfg4(a, dev, barrier):
    """BASELINE.json configs[4]: the two-field chaotic model at 512^3 and 1024^3, fp64 and fp32, order 2/4/6, 50
    steps each.  Initial conditions are generated on the device (pycool_init_fields: no 34 GB host arrays), so the
    cells carry no e2e; one JSON line per cell."""
    import torch
    from paper_1201_5029_b200 import binding, inputs
    steps = 50
    for name in ("cfg4_chaotic512", "cfg4_chaotic1024"):
        for precision in (64, 32):
            cfg = inputs.config(name)
            N, nf = cfg["N"], cfg["nfields"]
            for order in (2, 4, 6):
                lat = binding.from_config(cfg, device=dev, order=order, precision=precision)
                lat.init_fields(cfg["seed"], *inputs.spectra(cfg))
                lat.set_background(1.0)
                sampler = ClockSampler(dev.index or 0)
                sampler.start(); sampler.wait_first()
                lat.step(max(a.warmup, 3)); lat.sync()
                c0 = lat.launch_counts()
                ms = timed_steps(lat, steps, barrier, lat.stream)
                launches = sum(lat.launch_counts()) - sum(c0)
                roof = roofline_block(lat, name, precision, N, nf, steps, barrier)
                clocks = sampler.stop()
                line = {"metric": METRIC, "value": whole_job_value(N, nf, steps, 1, ms * 1e-3), "unit": UNIT, "n_gpus": 1,
                        "steps": steps, "warmup": max(a.warmup, 3), "ms_per_step": ms / steps, "higher_is_better": True,
                        "scaling": "weak", "vs_baseline": None, "dtype": "f%d" % precision, "data": "synthetic",
                        "config": {"workload": "%s: %d^3 x %d fields, model %d, order %d, dt=%g, %d-bit (sweep cell)"
                                   % (name, N, nf, cfg["model"], order, cfg["dt"], precision),
                                   "l2": "inputs larger than L2", "parallelism": "single GPU",
                                   "inputs": "pycool_init_fields (device-generated vacuum spectrum)"},
                        "clocks": clocks, "gpu_launches": launches, "roofline": roof, "a_final": lat.energies().a}
                print(json.dumps(line), flush=True)
                lat.close()
                del lat
                torch.cuda.empty_cache()


def main():
    a = parse()
    from paper_1201_5029_b200 import inputs
    cfg = inputs.config(a.workload)
    cfg["name"] = a.workload
    order = a.order or cfg["order"]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    N, nf = cfg["N"], cfg["nfields"]
    config = {"workload": "%s: %d^3 x %d fields, model %d, order %d, dt=%g, %d-bit" %
              (a.workload, N, nf, cfg["model"], order, cfg["dt"], a.precision),
              "l2": ("inputs larger than L2 (state %.1f GiB vs 126 MB)" if 2 * nf * N ** 3 * (a.precision // 8) > 126e6 else
                     "state %.3f GiB FITS in the 126 MB L2: the HBM roofline is not the yardstick for this workload")
                    % (2 * nf * N ** 3 * (a.precision // 8) / 2 ** 30),
              "parallelism": "replicas only" if a.gpus > 1 else "single GPU"}

    if a.impl == "reference":
        if rank != 0:
            return 0
        osteps = max(1, min(a.steps, 50))
        v, ms, sample = time_oracle(cfg, order, osteps, min(a.warmup, 1), a.precision)
        line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
                "warmup": a.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f%d" % a.precision, "data": "synthetic", "config": config,
                "cpu_baseline": cpu_baseline_block(v, sample),
                "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    import torch
    import torch.distributed as dist
    from paper_1201_5029_b200 import binding, build
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    if a.sweep:
        if rank == 0:
            sweep_cfg4(a, dev, barrier if world == 1 else (lambda: torch.cuda.synchronize(dev)))
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    if a.device_init:
        a.no_e2e = True
    else:
        phi, pi = inputs.make_initial(cfg, precision=a.precision)
        h_phi = torch.from_numpy(phi).pin_memory()
        h_pi = torch.from_numpy(pi).pin_memory()
        del phi, pi
    lat = binding.from_config(cfg, device=dev, order=order, precision=a.precision)
    if a.tile >= 0:
        lat.set_tile(a.tile)
    if a.zchunk > 0:
        lat.set_zchunk(a.zchunk)
    if a.item_order >= 0:
        lat.set_item_order(a.item_order)
    if a.persistent >= 0:
        lat.set_persistent(a.persistent)
    if a.cooperative >= 0:
        lat.set_cooperative(a.cooperative)
    if a.fused_tail >= 0:
        lat.set_fused_tail(a.fused_tail)
    if a.device_init:
        lat.init_fields(cfg["seed"], *inputs.spectra(cfg))
        config["inputs"] = "pycool_init_fields (device-generated)"
    else:
        lat.set_fields(h_phi, h_pi)
    lat.set_background(1.0)
    # clocks and throttle reasons are sampled from here (warm-up: the same steps as the timed region) to the end
    # of the timed region; nvidia-smi needs ~0.1 s to deliver its first line, the timed region may be shorter
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        sampler.wait_first()
    lat.step(a.warmup)
    lat.sync()

    # ---- device-resident timing: EXACTLY K steps between two events on the context stream, nothing else in the
    # stream (event records between launches would switch off the stage-to-stage launch overlap)
    c0 = lat.launch_counts()
    ms = timed_steps(lat, a.steps, barrier, lat.stream)
    c1 = lat.launch_counts()
    launches = sum(c1) - sum(c0)
    ms = max_over_ranks(ms, world, dev)
    value = whole_job_value(N, nf, a.steps, world, ms * 1e-3)

    # ---- roofline pass (per-launch CUDA events)
    roof = roofline_block(lat, a.workload, a.precision, N, nf, a.steps, barrier)
    clocks = sampler.stop() if rank == 0 else None
    lat.sync()

    # ---- row a7, on demand: pycool_energies (reads phi and pi once: 2 sizeof(real) bytes per field-site), wall
    # clock of the synchronising call, best of 3
    lat.energies()
    t_en = []
    for _ in range(3):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        lat.energies()
        t_en.append(time.perf_counter() - t0)
    en_ms = min(t_en) * 1e3

    # ---- SURVEY 8(f) rank 2, on demand: the workload's initial conditions generated on the device
    # (pycool_init_fields: spectrum fill + cuFFT Z2D + scatter per array), wall clock of the synchronising call
    init = None
    if N % 2 == 0 and not a.no_init:
        specs = inputs.spectra(cfg)
        lat.init_fields(cfg["seed"], *specs)                     # loads cuFFT, builds the plan once
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        lat.init_fields(cfg["seed"], *specs)
        init = {"ms": (time.perf_counter() - t0) * 1e3, "arrays": 2 * nf,
                "what": "pycool_init_fields: %d arrays of %d^3 (Philox + Box-Muller spectrum fill, cuFFT Z2D incl. "
                        "plan, scatter with ghost images), host wall clock; the host generator + H2D it replaces "
                        "is the set_fields leg of e2e plus the numpy FFTs" % (2 * nf, N)}

        lat.field_spectrum(0, 0)                                 # D2Z plan once
        t0 = time.perf_counter()
        lat.field_spectrum(0, 0)
        init["field_spectrum_ms"] = (time.perf_counter() - t0) * 1e3    # one array: gather + cuFFT D2Z + shell sums

    # ---- end to end: host buffers -> host buffers
    e2e = None
    if not a.no_e2e:
        esz = a.precision // 8
        barrier()
        t0 = time.perf_counter()
        lat.set_fields(h_phi, h_pi)
        lat.set_background(1.0)
        lat.step(a.steps)
        en = lat.energies()
        lat.read_fields(h_phi, h_pi)
        barrier()
        te = time.perf_counter() - t0
        te = max_over_ranks(te, world, dev)
        e2e = {"value": whole_job_value(N, nf, a.steps, world, te), "unit": UNIT, "h2d_bytes_per_step": 2 * nf * N ** 3 * esz / a.steps,
               "d2h_bytes_per_step": (2 * nf * N ** 3 * esz + 208) / a.steps,
               "what": "set_fields(H2D) + set_background + %d steps + energies + read_fields(D2H), pinned host buffers, "
                       "wall clock; bytes are per step of the %d-step job" % (a.steps, a.steps),
               "a_final": en.a}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peak, _ = measured_peaks()
    esz = a.precision // 8
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
            "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f%d" % a.precision, "data": "synthetic", "config": config, "clocks": clocks,
            "gpu_launches": launches, "roofline": roof}
    line["stage_su_per_s"] = value * {2: 1, 4: 3, 6: 7, 8: 15}[order]   # stage-normalised, SU/s x stages
    en_bytes = 2.0 * esz * N ** 3 * nf
    line["energies"] = {"ms": en_ms, "achieved": en_bytes / (en_ms * 1e-3) / 1e9, "unit": "GB/s",
                        "frac": en_bytes / (en_ms * 1e-3) / 1e9 / peak,
                        "what": "pycool_energies (sums of pi^2, G, phi D phi, V; reduce; D2H), host wall clock"}
    if init:
        line["init_fields"] = init
    if e2e:
        line["e2e"] = e2e
    if not a.no_linear and world == 1:
        line["linear"] = linear_block(dev)
    if not a.no_cpu_baseline and world == 1:
        stages = {2: 1, 4: 3, 6: 7, 8: 15}[order]
        v, _, sample = time_oracle(cfg, order, max(1, round(100 / stages)), 1, a.precision)     # ~13 s of CPU work
        line["cpu_baseline"] = cpu_baseline_block(v, sample)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
