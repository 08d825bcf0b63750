#!/usr/bin/env python
"""Writes tests/golden/full_length_<key>.json: the CPU oracle run over the FULL length of a
BASELINE.json config (final E, Q, KE, arrest count, the first arrests) on the seeded input of
paper_2603_24370_b200/workloads.py.  Calls only oracle/ and the input generators -- never the CUDA
path.  Hours of CPU time in total; run once per config:

    python tests/golden/make_full_length.py c2 c4 c5 c3l1 c3l2

keys: c1 (64^2, 1000 steps)  c2 (1024^2, 10000)  c3l1 / c3l2 (AH 2048^2, lambda 1 / 2, 20000)
      c4 (4096^2, 5000)  c5 (lattices 0, 101, 255 of the 256 x 256^2 sweep, 5000)
and, for the SURVEY 8(f) NEXT rows (not BASELINE configs; minutes of CPU time each):
      verlet (config 1's input, 1000 steps of the one-gradient-per-step integrator)
      d2d (128^2, the mirrored = antiskyrmion ansatz with the D2d DMI table, PAPER.md:141, 2000 steps)
      bs / bsbroken (baby Skyrme 128^2, standard / Z_3 broken potential, 2000 steps)
      demag (96^2, 2 Neel skyrmions, Neel DMI + demagnetising field g = 1, 300 Verlet steps)
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2603_24370_b200 import workloads as W  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
C5_LATTICES = (0, 101, 255)


def next_row_workload(key):
    """(workload, integrator) of the NEXT-row keys; tests/test_gpu_full_length.py builds the same."""
    if key == "verlet":
        return W.baseline_config(1), "verlet"
    if key == "d2d":
        w = W.cm_single(N=128, K=0.2, mirror=True, steps=2000)
        w.dmi = W.DMI_D2D
        return w, "rk4"
    if key == "bs":
        return W.bs_single(N=128, steps=2000), "rk4"
    if key == "bsbroken":
        return W.bs_single(N=128, pot=W.POT_BROKEN, potN=3, mu=0.8, steps=2000), "rk4"
    if key == "demag":
        # Neel skyrmions (the Bloch ansatz turned by 90 degrees about e3 in spin space: their
        # in-plane part is radial, so they carry magnetic charge; Bloch ones have div n = 0)
        w = W.cm_multi(N=96, count=2, margin=5.0, min_sep=6.0, steps=300)
        f = w.fields.copy()
        w.fields = np.ascontiguousarray(np.stack([-f[:, 1], f[:, 0], f[:, 2]], axis=1))
        w.demag, w.dmi, w.K = 1.0, W.DMI_NEEL, 0.1
        return w, "verlet"
    return None


def run(w, b, steps, log_every, integrator="rk4"):
    B = w.B if w.B_batch is None else float(w.B_batch[b])
    m = oracle.model(w.theory, w.Nx, w.Ny, w.h, kappa=w.kappa, B=B, K=w.K, lam=w.lam, dmi=w.dmi,
                     mu=w.mu, pot=w.pot, potN=w.potN, demag=w.demag)
    fl = oracle.Flow(m, w.dt, integrator=integrator)
    fl.set_fields(w.fields[b])
    E0, Q0 = fl.energy, fl.charge
    trace, done, t0 = [], 0, time.time()
    while done < steps:
        k = min(log_every, steps - done)
        fl.step(k)
        done += k
        s = fl.scalars()
        trace.append([done, s["E"], s["Q"], s["n_arrests"]])
        print(f"  {w.name}[{b}] step {done}/{steps} E={s['E']:.12g} Q={s['Q']:.9g} "
              f"arrests={s['n_arrests']} {time.time() - t0:.0f}s", flush=True)
    s = fl.scalars()
    _, _, de, _ = oracle.energy_charge(m, fl.get_fields()[0], densities=True)
    return {"lattice": b, "steps": steps, "E0": E0, "Q0": Q0, "E": s["E"], "Q": s["Q"],
            "KE": s["KE"], "n_arrests": s["n_arrests"], "arrests_first": fl.arrests()[:200],
            "abs_density_sum_h2": float(m.h * m.h * np.abs(de).sum()), "trace": trace,
            "cpu_seconds": time.time() - t0, "threads": oracle.threads()}


def main(keys):
    for key in keys:
        if key == "c1":
            w, lat = W.baseline_config(1), (0,)
        elif key == "c2":
            w, lat = W.baseline_config(2), (0,)
        elif key in ("c3l1", "c3l2"):
            w, lat = W.baseline_config(3, lam=1.0 if key == "c3l1" else 2.0), (0,)
        elif key == "c4":
            w, lat = W.baseline_config(4), (0,)
        elif key == "c5":
            w, lat = W.baseline_config(5), C5_LATTICES
        elif next_row_workload(key):
            (w, integ), lat = next_row_workload(key), (0,)
        else:
            raise SystemExit(f"unknown key {key}")
        if key in ("c1", "c2", "c3l1", "c3l2", "c4", "c5"):
            integ = "rk4"
        out = {"key": key, "workload": w.name, "Nx": w.Nx, "Ny": w.Ny, "h": w.h, "dt": w.dt,
               "kappa": w.kappa, "B": w.B, "K": w.K, "lambda": w.lam, "seed0": W.SEED0,
               "integrator": integ, "written_by": "tests/golden/make_full_length.py (oracle only)",
               "runs": [run(w, b, w.steps, max(1, w.steps // 20), integ) for b in lat]}
        with open(os.path.join(HERE, f"full_length_{key}.json"), "w") as f:
            json.dump(out, f, indent=1)
        print("wrote", key, flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["c1"])
