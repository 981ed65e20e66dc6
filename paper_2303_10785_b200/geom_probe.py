"""Two metrics_compute calls on the moving-mesh freestream workload (config 2 at n^3): the command the geometry
profiles under profiles/ were taken with (python -m paper_2303_10785_b200.geom_probe 256 under ncu)."""
import sys

import torch

import workloads as W
from paper_2303_10785_b200.binding import Grid


def main(n=256, reps=2):
    wl = W.c2_dynamic_freestream(n=n)
    g = Grid(wl, device=torch.device("cuda", 0))
    for r in range(3):
        g.metrics_compute(0.01 * (r + 1))
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for r in range(reps):
        g.metrics_compute(0.1 + 0.01 * r)
    e1.record()
    torch.cuda.synchronize()
    print("metrics_compute %d^3 moving: %.3f ms per call" % (n, e0.elapsed_time(e1) / reps))


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 256, int(sys.argv[2]) if len(sys.argv) > 2 else 2)
