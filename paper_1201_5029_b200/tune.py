"""In-process A/B of launch geometries of the fused drift+kick kernel on one lattice.

    python -m paper_1201_5029_b200.tune <workload> <precision> "zc,order[,tile];zc,order[,tile];..." [steps] [repeats]

For every geometry (z-chunk planes, item order as for pycool_set_item_order, optionally the kernel variant) the same
resident lattice is stepped `steps` times between two CUDA events, the geometries taken in turn `repeats` times, so
all of them see the same board state (boxes and power states differ by a few per cent between separate runs).
Initial conditions come from pycool_init_fields; throughput does not depend on the values.
"""
import statistics
import sys


def main(argv):
    import torch
    from . import binding, inputs
    wl, prec = argv[1], int(argv[2])
    geos = [tuple(int(x) for x in c.split(",")) for c in argv[3].split(";")]
    steps = int(argv[4]) if len(argv) > 4 else 20
    reps = int(argv[5]) if len(argv) > 5 else 4
    cfg = inputs.config(wl)
    lat = binding.from_config(cfg, precision=prec)
    lat.init_fields(cfg["seed"], *inputs.spectra(cfg))
    lat.set_background(1.0)
    res = {g: [] for g in geos}
    for _ in range(reps):
        for g in geos:
            if len(g) > 2:
                lat.set_tile(g[2])
            lat.set_zchunk(g[0])
            lat.set_item_order(g[1])
            lat.step(3)
            lat.sync()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(lat.stream)
            lat.step(steps)
            lat.flush()
            e1.record(lat.stream)
            torch.cuda.synchronize()
            res[g].append(e0.elapsed_time(e1) / steps)
    stages = {2: 1, 4: 3, 6: 7, 8: 15}[cfg["order"]]
    for g in geos:
        v = res[g]
        print("%s fp%d zc %d order %d%s: ms/step median %.4f min %.4f max %.4f, %.2f us per stage" %
              (wl, prec, g[0], g[1], (" variant %d" % g[2]) if len(g) > 2 else "", statistics.median(v), min(v), max(v),
               statistics.median(v) / stages * 1e3))


if __name__ == "__main__":
    main(sys.argv)
