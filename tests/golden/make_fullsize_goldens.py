#!/usr/bin/env python
"""Writes tests/golden/full_<config>_<phase><step>.txt: psi of the CPU ORACLE at sampled grid points, plus norm,
mu, E and rms, for BASELINE.json's configs at their FULL sizes (parity-window table).

    python tests/golden/make_fullsize_goldens.py C4          # 512^3 imaginary time, checkpoints 1, 10
    python tests/golden/make_fullsize_goldens.py C5          # 768x768x384 real time, checkpoints 1, 10, 50, 100
    python tests/golden/make_fullsize_goldens.py C3          # 256^3: relaxation 1, 100, 200, 300; quench after 200 and 300
    python tests/golden/make_fullsize_goldens.py C2          # 128^3 imaginary time, checkpoints 1, 100, 350

This script calls ONLY oracle/ (the plain C oracle through its ctypes binding) and the seeded input
generator paper_1610_05329_b200/inputs.py (which holds none of the method's arithmetic).  It never loads the
CUDA library.  It is run offline, once, on host cores (the oracle needs 1.5-4 minutes per step at these sizes);
tests/test_gpu_fullsize_goldens.py replays the same dgpe_step calls on the GPU and compares.

File format (text): '# key: value' header lines, then one row per sampled point:  i j k Re(psi) Im(psi)
(%.17g: round-trip exact).  Sample points: structured points (corners, face centres, the centre and its
neighbours, the first/last interior nodes, lines through the centre), seeded random points in the central
region where psi is not negligible, seeded random points anywhere in the box, and the 64 points of largest
|psi| at that checkpoint.
"""
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import binding as ob                      # noqa: E402
from paper_1610_05329_b200 import inputs              # noqa: E402   (seeded inputs only)

N_CENTRAL, N_ANYWHERE, N_TOP = 640, 256, 64


def sample_points(cfg, psi):
    nx, ny, nz = cfg.shape
    n = np.array(cfg.shape)
    c = n // 2
    pts = []
    for i in (0, nx - 1):
        for j in (0, ny - 1):
            for k in (0, nz - 1):
                pts.append((i, j, k))                                   # corners
    for a in range(3):
        for v in (0, 1, n[a] - 2, n[a] - 1):                            # faces and first/last interior planes
            p = list(c)
            p[a] = v
            pts.append(tuple(p))
    pts.append((1, 1, 1))
    pts.append((nx - 2, ny - 2, nz - 2))
    for di in (-1, 0, 1):
        for dj in (-1, 0, 1):
            for dk in (-1, 0, 1):
                pts.append((c[0] + di, c[1] + dj, c[2] + dk))            # the centre and its 26 neighbours
    for a in range(3):                                                  # a line through the centre along each axis
        for v in range(0, n[a], max(1, n[a] // 64)):
            p = list(c)
            p[a] = v
            pts.append(tuple(p))
    # seeded random points: central region (half-width 3.5 standard deviations of the initial |psi|^2 ... of psi0)
    cnt = np.arange(3 * (N_CENTRAL + N_ANYWHERE), dtype=np.uint64)
    u = inputs.uniform01(cfg.seed, 20, cnt).reshape(-1, 3)
    half = np.array([min(n[a] // 2 - 1, int(np.ceil(3.5 / np.sqrt(cfg.gauss[a]) / cfg.d[a]))) for a in range(3)])
    cen = c + np.floor((2.0 * u[:N_CENTRAL] - 1.0) * (half + 0.5)).astype(np.int64)
    anyw = np.floor(u[N_CENTRAL:] * n).astype(np.int64)
    for p in np.concatenate([cen, anyw]):
        pts.append(tuple(int(v) for v in np.clip(p, 0, n - 1)))
    # the points of largest |psi| at this checkpoint
    mag = (psi.real ** 2 + psi.imag ** 2).ravel()
    top = np.argpartition(mag, mag.size - N_TOP)[-N_TOP:]
    for lin in np.sort(top):
        pts.append(tuple(int(v) for v in np.unravel_index(int(lin), cfg.shape)))
    seen, out = set(), []
    for p in pts:
        if p not in seen:
            seen.add(p)
            out.append(p)
    return np.array(out, dtype=np.int64)


def write_checkpoint(tag, cfg, O, psi, phase, step, psi0_sha, call, extra=None):
    t0 = time.perf_counter()
    pts = sample_points(cfg, psi)
    obs = {"norm": O.norm(psi), "mu": O.chempot(psi), "energy": O.energy(psi)}
    rms = O.rms(psi)
    path = os.path.join(HERE, f"full_{tag}_{phase}{step:04d}.txt")
    with open(path, "w") as f:
        f.write(f"# written by: tests/golden/make_fullsize_goldens.py {tag}  (oracle/ only; never the CUDA path)\n")
        f.write(f"# config: {cfg.name}\n")
        f.write(f"# create_args: {' '.join(repr(v) for v in cfg.create_args())}\n")
        f.write(f"# seed: {cfg.seed}\n")
        f.write(f"# psi0_sha256: {psi0_sha}\n")
        f.write(f"# call: {call}\n")
        f.write(f"# phase: {phase}\n")
        f.write(f"# step: {step}\n")
        for k, v in obs.items():
            f.write(f"# {k}: {v:.17g}\n")
        f.write("# rms: " + " ".join(f"{v:.17g}" for v in rms) + "\n")
        f.write(f"# max_abs_psi: {float(np.sqrt(np.max(psi.real ** 2 + psi.imag ** 2))):.17g}\n")
        for k, v in (extra or {}).items():
            f.write(f"# {k}: {v}\n")
        f.write(f"# npoints: {len(pts)}\n")
        for (i, j, k) in pts:
            v = psi[i, j, k]
            f.write(f"{i} {j} {k} {v.real:.17g} {v.imag:.17g}\n")
    print(f"[{tag}] wrote {os.path.basename(path)}: norm={obs['norm']:.15g} mu={obs['mu']:.15g} E={obs['energy']:.15g} "
          f"rms={rms} ({time.perf_counter() - t0:.0f} s for observables)", flush=True)


def run_steps(O, psi, upto, done, tag, times):
    while done < upto:
        t0 = time.perf_counter()
        rc = O.step(psi, 1)
        dt = time.perf_counter() - t0
        times.append(dt)
        done += 1
        print(f"[{tag}] step {done}: rc={rc} {dt:.1f} s", flush=True)
        if rc != ob.OK:
            raise SystemExit(f"[{tag}] oracle status {rc} at step {done}")
    return done


def timing_note(times):
    s = sorted(times)
    return {"oracle_s_per_step_median": f"{s[len(s) // 2]:.2f}", "oracle_s_per_step_min": f"{s[0]:.2f}",
            "oracle_steps_timed": len(s), "oracle_cores": 1}


def simple(tag, checkpoints):
    """psi0 -> one handle, checkpoints along one trajectory (C2, C4, C5)."""
    cfg = inputs.CONFIGS[tag]
    psi = inputs.initial_state(cfg)
    sha = hashlib.sha256(psi.tobytes()).hexdigest()
    O = ob.Oracle(*cfg.create_args())
    phase = "imag" if cfg.mode == inputs.IMAG else "real"
    write_checkpoint(tag, cfg, O, psi, phase, 0, sha, "initial state (inputs.initial_state)")
    done, times = 0, []
    for cp in checkpoints:
        done = run_steps(O, psi, cp, done, tag, times)
        write_checkpoint(tag, cfg, O, psi, phase, cp, sha, f"odgpe_step from psi0, {cp} steps in all", timing_note(times))


def c3():
    """BJ:configs[2] at 256^3: relaxation (imaginary time, g = 80, gdd = 40) with checkpoints 1, 100, 200, 300;
    real time after the quench to g = 64 (a) from the step-200 state (inside the smooth window):
    real steps 1, 10, 100; (b) from the step-300 state, the literal protocol (in the collapse): real steps 1, 10."""
    cfg = inputs.CONFIGS["C3"]
    relax = cfg.relax
    psi = inputs.initial_state(relax)
    sha = hashlib.sha256(psi.tobytes()).hexdigest()
    Oi, Or = ob.Oracle(*relax.create_args()), ob.Oracle(*cfg.create_args())
    write_checkpoint("C3", relax, Oi, psi, "relax", 0, sha, "initial state (inputs.initial_state)")
    # the real-time handle on the seeded Gaussian itself
    q = psi.copy()
    times_r = []
    run_steps(Or, q, 1, 0, "C3 real-from-psi0", times_r)
    write_checkpoint("C3", cfg, Or, q, "real0from0_", 1, sha, "real handle (g = 64), 1 step from psi0", timing_note(times_r))
    done, times = 0, []
    for cp in (1, 100, 200, 300):
        done = run_steps(Oi, psi, cp, done, "C3 relax", times)
        write_checkpoint("C3", relax, Oi, psi, "relax", cp, sha, f"imaginary handle (g = 80), {cp} steps from psi0",
                         timing_note(times))
        if cp in (200, 300):
            q = psi.copy()
            d2 = 0
            for rcp in ((1, 10, 100) if cp == 200 else (1, 10)):
                d2 = run_steps(Or, q, rcp, d2, f"C3 real after {cp}", times_r)
                write_checkpoint("C3", cfg, Or, q, f"quench{cp}real", rcp, sha,
                                 f"imaginary handle {cp} steps from psi0, then real handle (g = 64) {rcp} steps",
                                 timing_note(times_r))


if __name__ == "__main__":
    which = sys.argv[1] if len(sys.argv) > 1 else "C4"
    if which == "C4":
        simple("C4", [1, 10])
    elif which == "C5":
        simple("C5", [int(v) for v in sys.argv[2:]] or [1, 10, 50, 100])
    elif which == "C2":
        simple("C2", [1, 100, 350])
    elif which == "C3":
        c3()
    else:
        raise SystemExit("usage: make_fullsize_goldens.py C2|C3|C4|C5")
