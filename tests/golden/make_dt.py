"""Writes tests/golden/dt.json: the time step of each bench-size config, Eq. B.2 / B.3 evaluated by the
CPU ORACLE on the initial state (CFL as in the config).  Calls only oracle/ and the seeded input generators.

    python tests/golden/make_dt.py
"""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))
import workloads as W  # noqa: E402
from oracle import meg6_oracle as O  # noqa: E402


def main():
    out = {}
    for wl in (W.c1_vortex(n=32), W.c2_dynamic_freestream(n=64), W.c3_tgv(n=128)):
        g = O.Grid(wl)
        g.metrics_compute(wl["t0"])
        out[wl["name"]] = g.cfl_dt(wl["U0"], wl["cfl"])
        print(wl["name"], out[wl["name"]])
    with open(os.path.join(HERE, "dt.json"), "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
