#!/usr/bin/env python
"""bench.py -- throughput of the full SSCN step (BASELINE.json metric: fp64 SSCN steps/s and grid-point
updates/s at 512^3 on one B200; HBM GB/s vs peak).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl reference]

One "step" = one pass of the whole hot path (kernels K1..K8, the z sweep K8 fused into K5 when the z-line
kernels apply) over the psi of the
workload.  N = 1 times BASELINE.json's headline configuration C4 (512^3, imaginary time).  N > 1
(torchrun, one rank per GPU) runs N independent replicas -- the path does not shard without all-to-all
transposes -- and reports all ranks' steps over the slowest rank's time.
Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle instead (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sscn_steps_per_s"
UNIT = "steps/s"
# the oracle takes ~200 s per 512^3 step on one core (measured offline: tests/golden/full_C4_imag0010.txt,
# BASELINE.md section 3), so its legs in this script run a bounded sample of the workload:
# the same physics (spacings, dt, trap, g, gdd, seeded state recipe) on a smaller centred box
CPU_SAMPLE_BASELINE = (256, 256, 128)    # cpu_baseline leg: one step, ~10 s
CPU_SAMPLE_REFERENCE = (128, 128, 128)   # --impl reference: every step, ~2 s each
REPS = 3                                 # timed repetitions of K steps; the median is reported
CALL_STEPS = 10                          # steps per dgpe_step call inside a repetition (each call starts from psi0)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--rpsi", action="store_true",
                    help="imaginary-time configs: time the real-valued-psi path DGPE_IMAG_RPSI (SURVEY 8f NEXT-2); "
                         "not the headline, which stays complex psi as BASELINE.json states")
    ap.add_argument("--opt", default="", help="dgpe_create_ex options for A/B runs, e.g. 'fused_fft=0,tma=0' (include/dgpe.h)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload_name(cfg, rpsi=False):
    nx, ny, nz = cfg.shape
    mode = "imaginary-time" if cfg.mode == 0 else "real-time"
    src = (f"BASELINE.json configs[{int(cfg.name[1]) - 1}]" if cfg.name[0] == "C" else
           "grid of the paper's timing table " + cfg.name[1] + ", physics borrowed from C4: context only")
    kind = "fp64 REAL-valued psi (DGPE_IMAG_RPSI, SURVEY 8f NEXT-2; same step, 8 bytes per point)" if rpsi else "fp64 complex"
    return (f"{cfg.name}: {mode} dipolar GPE {nx}x{ny}x{nz} {kind}, dx={cfg.d[0]} dt={cfg.dt} "
            f"trap={cfg.trap} g={cfg.g} gdd={cfg.gdd} ({src})")


def l2_note(psi_bytes, spec_bytes):
    """How the timed steps stand to the 126 MB L2 (timing rule: say which)."""
    sizes = "psi %.3f GB + half-spectrum %.3f GB vs 126 MB" % (psi_bytes * 1e-9, spec_bytes * 1e-9)
    if psi_bytes + spec_bytes > 2 * 126e6:
        return "inputs larger than L2: " + sizes
    return ("working set NOT larger than L2 (" + sizes + "), no flush between steps: each step consumes the previous step's "
            "output, so L2 residency is part of this small workload; read steps/s, not the DRAM fractions")


def load_peaks():
    """Measured roofline denominators (driver-written); else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for nme, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_time(cfg, sample_shape, steps, warmup=0):
    """Seconds per oracle step on a `sample_shape` box with cfg's physics; returns (s/step, npoints)."""
    from oracle import binding as ob
    from paper_1610_05329_b200 import inputs
    sub = inputs.scaled(cfg, sample_shape)
    psi = inputs.initial_state(sub)
    O = ob.Oracle(*sub.create_args())
    if warmup:
        O.step(psi, warmup)
    t0 = time.perf_counter()
    O.step(psi, steps)
    dt = time.perf_counter() - t0
    return dt / steps, sub.npoints


def measured_full_size(cfg):
    """Seconds per oracle step at the FULL size of cfg, measured offline when tests/golden/make_fullsize_goldens.py wrote the
    goldens (recorded in their headers); None if there is no such record."""
    import glob
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "tests", "golden", f"full_{cfg.name}_*.txt"))):
        with open(path) as f:
            for line in f:
                if not line.startswith("#"):
                    break
                if line.startswith("# oracle_s_per_step_median:"):
                    best = float(line.split(":")[1])
    return best


def cpu_baseline(cfg, sample_shape, steps=1):
    s_per_step, npts = oracle_time(cfg, sample_shape, steps)
    pts_per_s = npts / s_per_step
    return {"value": pts_per_s / cfg.npoints, "unit": UNIT, "cores": 1, "kind": "oracle",
            "grid_pt_updates_per_s": pts_per_s,
            "measured_full_size_s_per_step": measured_full_size(cfg),
            "measured_full_size_note": "one core, offline, on the build container's host while the goldens were written "
                                       "(tests/golden/full_*.txt headers); not this box",
            "sample": (f"{steps} oracle step(s) of {cfg.name}'s physics on a {'x'.join(map(str, sample_shape))} box "
                       f"({npts / cfg.npoints:.4f} of the points), {s_per_step:.2f} s/step on 1 core of "
                       f"{os.cpu_count()}; value = sample grid-pt updates/s / {cfg.npoints} points")}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    s_per_step, npts = oracle_time(cfg, CPU_SAMPLE_REFERENCE, args.steps, args.warmup)
    pts_per_s = npts / s_per_step
    value = pts_per_s / cfg.npoints
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "grid_pt_updates_per_s": pts_per_s,
        "config": {"workload": workload_name(cfg), "sample_box": list(CPU_SAMPLE_REFERENCE)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": (f"each step = one oracle step of {cfg.name}'s physics on a "
                                    f"{'x'.join(map(str, CPU_SAMPLE_REFERENCE))} box, {s_per_step:.2f} s/step, scaled by "
                                    f"points to the {cfg.npoints}-point workload")},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
def ncu_traffic(kernel_name, rpsi=False):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the dominant kernel from
    the committed `ncu --set full` capture, recorded in profiles/traffic.csv (traffic_rpsi.csv for the
    real-valued path); else None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic_rpsi.csv" if rpsi else "traffic.csv")) as f:
            for line in f:
                name, _, rest = line.rstrip("\n").partition(",")
                if name == kernel_name:
                    return float(rest.split(",")[0])
    except Exception:
        pass
    return None


def run_b200(args, cfg):
    import torch
    from paper_1610_05329_b200 import binding, inputs, replicas
    from dataclasses import replace

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    rank, local_rank, world = replicas.init()
    torch.cuda.set_device(local_rank)
    K, W = args.steps, max(args.warmup, 3)
    mycfg = replace(cfg, seed=replicas.replica_seed(cfg.seed, rank))       # each replica: its own seeded state

    rpsi = bool(args.rpsi)
    if rpsi and cfg.mode != 0:
        raise SystemExit("--rpsi needs an imaginary-time config")
    G = binding.Dgpe(*mycfg.create_args()[:-1], binding.IMAG_RPSI if rpsi else mycfg.mode,
                     options=binding.parse_options(args.opt))
    state = inputs.initial_state(mycfg)
    if rpsi:
        import numpy as np
        state = np.ascontiguousarray(state.real)          # the imaginary-time initial states are real
    psi_host = torch.from_numpy(state).pin_memory()
    del state
    psi0 = psi_host.cuda()
    psi = psi0.clone()

    # ---- device-resident timing: inputs in HBM when the timed region starts ----
    # REPS repetitions of EXACTLY K steps each.  A repetition is made of dgpe_step calls of at most CALL_STEPS steps,
    # each starting again from psi0 (the restoring copy is outside the timed events), so that the literal C4 stays
    # inside its smooth window (NaN from step ~19) and every call returns status 0.  Each
    # repetition is bracketed by a barrier and a device synchronisation, timed with CUDA events on the stream the
    # kernels run on, and its duration is the MAX over ranks; the line reports the MEDIAN repetition.
    calls = [CALL_STEPS] * (K // CALL_STEPS) + ([K % CALL_STEPS] if K % CALL_STEPS else [])
    G.step(psi, W)
    psi.copy_(psi0)
    torch.cuda.synchronize()
    replicas.barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    rep_sec, status = [], 0
    for _ in range(REPS):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in calls]
        torch.cuda.synchronize()
        replicas.barrier()
        for (e0, e1), n in zip(evs, calls):
            psi.copy_(psi0)
            e0.record()
            rc = G.step(psi, n)
            e1.record()
            status = status or int(rc)
        torch.cuda.synchronize()
        replicas.barrier()
        sec_local = sum(e0.elapsed_time(e1) for e0, e1 in evs) * 1e-3
        _, sec = replicas.aggregate_throughput(K, sec_local)             # max over ranks
        rep_sec.append(sec)
    clocks = sampler.stop() if rank == 0 else None
    sec = sorted(rep_sec)[len(rep_sec) // 2]
    value = world * K / sec
    sec_local = sec
    finite = bool(torch.isfinite(psi if rpsi else torch.view_as_real(psi)).all())

    # the same shape with the dipolar strength reduced so that eps_dd < 1 (no collapse: SURVEY 8(d) "stable sibling"):
    # backs the statement that the timing does not depend on the data
    sibling = None
    if cfg.name == "C4" and world == 1 and not rpsi:
        Gs = binding.Dgpe(*replace(mycfg, gdd=60.0).create_args(), options=binding.parse_options(args.opt))
        psi.copy_(psi0)
        Gs.step(psi, 3)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        rc = Gs.step(psi, K)
        e1.record()
        torch.cuda.synchronize()
        sibling = {"gdd": 60.0, "steps_in_one_call": K, "status": int(rc), "ms_per_step": e0.elapsed_time(e1) / K}
        Gs.close()

    # ---- per-kernel durations, CUDA events on the handle's stream (dgpe_step_profile) ----
    psi.copy_(psi0)
    G.step_profile(psi, 2)
    psi.copy_(psi0)
    prof = G.step_profile(psi, min(K, 8))
    peak, peak_src = load_peaks()
    kernels = [{"name": n, "bytes": b, "ms": ms, "GBps": b / ms * 1e-6} for n, b, ms in prof]
    top = max(kernels, key=lambda k: k["ms"])
    step_ms = sec_local / K * 1e3
    roofline = {"bound": "hbm", "kernel": top["name"], "achieved": top["GBps"], "peak": peak, "unit": "GB/s",
                "frac": top["GBps"] / peak, "traffic": ncu_traffic(top["name"], rpsi) if cfg.name == "C4" else None,
                "traffic_source": ("committed ncu --set full capture of this kernel at C4 (profiles/traffic_rpsi.csv)" if rpsi else
                                   "committed ncu --set full capture of this kernel at C4 (profiles/traffic.csv)") if cfg.name == "C4"
                                  else None,
                "timing_source": "live: CUDA events between the kernels of dgpe_step_profile on the handle's stream",
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": top["bytes"], "kernel_ms": top["ms"],
                "share_of_step": top["ms"] / sum(k["ms"] for k in kernels)}
    step_gbps = G.bytes_per_step / step_ms * 1e-6
    built = sum(k["bytes"] for k in kernels)
    whole = {"algorithmic_bytes_per_step": G.bytes_per_step, "achieved": step_gbps, "frac": step_gbps / peak,
             "unit": "GB/s", "model": ("M1r = 72N + 8S (real-valued psi: SURVEY section 8f NEXT-2; DESIGN.md section 7)" if rpsi
                                        else "M1 = 144N + 8S (SURVEY section 8d; DESIGN.md section 7)"),
             "frac_of_nominal_8TBps": step_gbps / 8000.0,
             "as_built": {"bytes_per_step": built, "achieved": built / step_ms * 1e-6,
                          "frac": built / step_ms * 1e-6 / peak,
                          "model": "sum of the kernels' own algorithmic bytes (M2 = 112N + 8S when the z sweep is "
                                   "fused into K5)"}}

    # ---- end to end through the C-ABI with HOST buffers (dgpe_step_host) ----
    # the same K steps as calls of <= CALL_STEPS steps, each call = H2D of psi0 from pinned memory, the steps, D2H of the
    # result; wall clock around the (synchronous) calls, max over ranks, median of REPS repetitions
    e2e = None
    if not args.no_e2e:
        work = psi_host.clone().pin_memory()
        G.step_host(work, 1)                      # allocates the staging buffer, warms the copies
        nbytes = work.numel() * work.element_size()
        e2e_rep, e2e_status = [], 0
        for _ in range(REPS):
            torch.cuda.synchronize()
            replicas.barrier()
            t_rep = 0.0
            for n in calls:
                work.copy_(psi_host)              # restore the host state: not timed
                t0 = time.perf_counter()
                rc = G.step_host(work, n)         # H2D + n steps + D2H, returns after the stream is idle
                t_rep += time.perf_counter() - t0
                e2e_status = e2e_status or int(rc)
            replicas.barrier()
            _, t_max = replicas.aggregate_throughput(K, t_rep)
            e2e_rep.append(t_max)
        t_med = sorted(e2e_rep)[len(e2e_rep) // 2]
        e2e = {"value": world * K / t_med, "unit": UNIT, "h2d_bytes_per_step": nbytes * len(calls) / K,
               "d2h_bytes_per_step": nbytes * len(calls) / K,
               "call": f"dgpe_step_host(psi_pinned, n) for n in {calls}: each call one H2D of psi ({nbytes} B), n steps, one "
                       f"D2H; bytes per step = bytes per call x {len(calls)} calls / {K} steps",
               "ms_per_step": t_med / K * 1e3, "reps_ms_per_step": [t / K * 1e3 for t in e2e_rep], "status": e2e_status}
        del work

    if rank != 0:
        replicas.shutdown()
        return
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": sec / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "grid_pt_updates_per_s": value * cfg.npoints,
        "config": {"workload": workload_name(cfg, rpsi), "parallelism": f"replicas x{world} (no sharding, no collectives)",
                   "l2": l2_note(cfg.npoints * (8 if rpsi else 16), cfg.shape[0] * cfg.shape[1] * (cfg.shape[2] // 2 + 1) * 16),
                   "status": int(status), "finite": finite,
                   "timed": f"median of {REPS} repetitions of {K} steps; a repetition = dgpe_step calls of {calls} steps, each "
                            f"from psi0 (restoring copy untimed), CUDA events on the kernels' stream, max over ranks",
                   "note": "literal C4 is in the dipolar-collapse regime (NaN from step ~19, DESIGN.md section 4): calls of "
                           "<= 10 steps stay inside its smooth window, status 0"},
        "reps_ms_per_step": [t / K * 1e3 for t in rep_sec],
        "spread": (max(rep_sec) - min(rep_sec)) / sec,
        "clocks": clocks,
        # kernels launched inside one timed repetition: per call one k_set_scal, per step the step's kernels, and in
        # imaginary time k_scale + k_set_scal at the end of each call
        "gpu_launches": K * G.launches_per_step + len(calls) * (3 if cfg.mode == 0 else 1),
        "roofline": roofline, "step_roofline": whole, "kernels": kernels,
    }
    if sibling is not None:
        line["stable_sibling"] = sibling
    if e2e is not None:
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg, CPU_SAMPLE_BASELINE)
    print(json.dumps(line), flush=True)
    replicas.shutdown()


def main():
    args = parse()
    from paper_1610_05329_b200 import inputs
    cfg = inputs.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_b200(args, cfg)


if __name__ == "__main__":
    main()
