"""Board power and SM clock while spills run back to back (measurement tool; profiles/r2_response_bound.md cites it).

    python -m paper_2212_09807_b200.measure_power [config] [spills]

Runs `spills` whole-spill passes of BASELINE configs[config] (default 3, 12) through lartpc_run_spill with nvidia-smi sampling
clocks.sm, power.draw (averaged by the driver) and power.draw.instant beside it (the driver refreshes them about every
100 ms, whatever the sampling period), and prints their distributions.  Nothing here touches the clocks."""
import subprocess
import sys
import time

import numpy as np


def main(argv):
    import torch
    from . import lartpc, workloads as W
    cfg = int(argv[1]) if len(argv) > 1 else 3
    n_spills = int(argv[2]) if len(argv) > 2 else 12
    wl = W.make_config(cfg)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    seg = sim.upload_segments(wl.segments)
    cap = int(8 * wl.n_segments) + 4096
    sim.run_spill(seg, wl.seed, hit_capacity=cap)                      # warm-up: buffers sized, hints set
    torch.cuda.synchronize()
    smi = subprocess.Popen(["nvidia-smi", "-i", str(torch.cuda.current_device()),
                            "--query-gpu=clocks.sm,power.draw,power.draw.instant,power.limit",
                            "--format=csv,noheader,nounits", "-lms", "20"], stdout=subprocess.PIPE, text=True)
    time.sleep(0.5)
    t0 = time.time()
    for _ in range(n_spills):
        sim.run_spill(seg, wl.seed, hit_capacity=cap)
    torch.cuda.synchronize()
    wall = time.time() - t0
    smi.terminate()
    rows = []
    for line in smi.stdout.read().strip().splitlines():
        try:
            rows.append([float(x) for x in line.split(",")])
        except ValueError:
            pass
    rows = np.array(rows[25:])                                         # (the half second before the first spill)
    if len(rows) == 0:
        print("no samples")
        return 1
    pct = [5, 25, 50, 75, 95]
    print("configs[%d]: %d spills in %.2f s (%.1f ms each), %d samples, power limit %.0f W" % (
        cfg, n_spills, wall, 1e3 * wall / n_spills, len(rows), rows[:, 3].max()))
    print("SM clock MHz, percentiles %s: %s" % (pct, np.percentile(rows[:, 0], pct).round(0).tolist()))
    print("power.draw W (driver average): %s" % np.percentile(rows[:, 1], pct).round(0).tolist())
    print("power.draw.instant W: %s" % np.percentile(rows[:, 2], pct).round(0).tolist())
    sim.close()
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
