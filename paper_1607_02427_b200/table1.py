"""Table-I-like sweep: particle-timesteps/s of dem_step for spheres, triangular plates, cubes and icosahedra at
N = 256, 4096, 65536 (Table I and Figure 4).

    python -m paper_1607_02427_b200.table1 [--equil 2000] [--steps 500] [--shapes sphere,cube] [--sizes 256,4096]

The paper's states (thermalised dense fluids of unstated density and rounding radius) are not available; the start
states are dem_inputs.table1_state (seeded lattices, kT = 1), equilibrated here with --equil NVE steps before --steps
timed ones.  FP32 context, the library's defaults (exact culling on), device-resident arrays, neighbour rebuilds
included, CUDA events on the launching stream.  Prints one markdown table; the paper's GPU column (Quadro M6000,
another machine and other densities) is context, not a like-for-like comparison.  Runs on the CUDA library only.
"""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import dem_inputs as di  # noqa: E402

# Table I, PAPER.md:101-109 (PTPS_GPU on a Quadro M6000); plates appear only in Figure 4 (no numbers printed)
PAPER_GPU_PTPS = {("sphere", 256): 3.0e6, ("sphere", 4096): 4.6e7, ("sphere", 65536): 1.59e8,
                  ("cube", 256): 1.9e5, ("cube", 4096): 3.8e5, ("cube", 65536): 3.5e5,
                  ("icosahedron", 256): 6.0e4, ("icosahedron", 4096): 8.0e4, ("icosahedron", 65536): 6.9e4}
SKIN = {"sphere": 0.3, "plate": 0.2, "cube": 0.3, "icosahedron": 0.15}


def run_one(pkg, shape, n, equil, steps, seed=0):
    import torch

    st = di.table1_state(shape, n, seed)
    dem, t = pkg.from_state(st, "f32")
    f = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    tq = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    args = (t["pos"], t["quat"], t["vel"], t["angmom"], t["shape_id"], st["box"], st["dt"])
    skin = SKIN[shape]
    dem.step(*args, equil, skin, f, tq)
    e0 = dem.energy(t["quat"], t["vel"], t["angmom"], t["shape_id"], f)
    l0 = dem.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    dem.step(*args, steps, skin, f, tq)
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1)
    e1 = dem.energy(t["quat"], t["vel"], t["angmom"], t["shape_id"], f)
    counts, _ = dem.get_neighbors()
    cnt = dem.get_counters()
    row = dict(shape=shape, N=n, neighbours=float(counts.float().mean()), ms_per_step=ms / steps,
               ptps=n * steps / (ms * 1e-3), u_per_n=e1[0] / n, kT=2.0 * e1[1] / (3.0 * n),
               drift=abs(e1.sum() - e0.sum()) / n, active_terms=int(cnt["active"]), degenerate=int(cnt["degenerate"]),
               launches_per_step=(dem.launch_count() - l0) / steps, paper_gpu=PAPER_GPU_PTPS.get((shape, n)))
    dem.close()
    return row


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--equil", type=int, default=2000)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--shapes", default=",".join(di.TABLE1_SHAPES))
    ap.add_argument("--sizes", default=",".join(str(k) for k in sorted(di.TABLE1_CELLS)))
    a = ap.parse_args(argv)
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("table1 needs a CUDA device: the product has no CPU path")
    import paper_1607_02427_b200 as pkg

    print("| shape | N | neighbours / particle | U/N | kT (translation) | ms / step | launches / step | PTPS (B200, this library) "
          "| PTPS_GPU of Table I (M6000; context) | drift / N over the timed steps |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    rows = []
    for shape in a.shapes.split(","):
        for n in (int(x) for x in a.sizes.split(",")):
            r = run_one(pkg, shape, n, a.equil, a.steps)
            rows.append(r)
            assert r["degenerate"] == 0 and np.isfinite(r["drift"]), r
            print("| %s | %d | %.1f | %.3f | %.3f | %.4f | %.1f | %.3g | %s | %.1e |" % (
                shape, n, r["neighbours"], r["u_per_n"], r["kT"], r["ms_per_step"], r["launches_per_step"], r["ptps"],
                ("%.3g" % r["paper_gpu"]) if r["paper_gpu"] else "—", r["drift"]), flush=True)
    return rows


if __name__ == "__main__":
    main()
