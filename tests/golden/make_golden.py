"""Writes tests/golden/<key>.json: observables of a full BASELINE.json run computed by the CPU oracle.

    python tests/golden/make_golden.py C1 C2 C3 [C4 C5] [X0 X1 X2]

C1-C5 are the BASELINE.json configs; X0-X2 the remaining program variants of PAPER.md:15 (imag2dXY,
imag2dXZ, real2dXZ; inputs.py).

Calls only oracle/ (the plain fp64 CPU implementation written from the paper under the readings of
DESIGN.md) and the seeded input generator; nothing from the CUDA path.  These are NOT values printed
in the paper (PAPER.md prints none); they let the GPU tests check the 1e-9 full-run bar of
BASELINE.json on configs whose oracle run takes tens of minutes.
"""
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import binding as ob                                     # noqa: E402
from paper_1601_04640_b200.inputs import initial_psi, workload      # noqa: E402


def run(key):
    w = workload(key)
    o = ob.Oracle(ob.params_of(w))
    o.set_psi(initial_psi(w))
    if (w.G_run, w.D_run) != (w.G, w.D):
        o.set_coupling(w.G_run, w.D_run)          # reading S18: quench before the first step
    rows = [{"step": 0, **o.observables()}]
    t0 = time.time()
    done = 0
    while done < w.steps:
        n = min(w.report_every, w.steps - done)
        o.step(n)
        done += n
        rows.append({"step": done, **o.observables()})
        print(f"{key} step {done}/{w.steps}  {time.time() - t0:.0f}s  mu={rows[-1]['mu']:.12f}", flush=True)
    out = {"workload": key, "name": w.name, "source": "oracle/dbec_oracle.cpp via tests/golden/make_golden.py",
           "G_run": w.G_run, "D_run": w.D_run, "steps": w.steps, "oracle_threads": ob.threads(),
           "observables": rows}
    with open(os.path.join(HERE, f"{key}.json"), "w") as f:
        json.dump(out, f, indent=1)
    o.close()


if __name__ == "__main__":
    for k in sys.argv[1:]:
        run(k)
