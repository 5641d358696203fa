"""Short-term energy conservation against the timestep (Fig. 3): the standard
deviation of the total energy per particle, sigma(E/N), recorded at high frequency over an NVE run of duration 10 tau,
for squares (2D) and tetrahedra (3D), with DEM_F32 and DEM_F64 contexts, as a function of dt.

    python -m paper_1607_02427_b200.fig3 [--duration 10] [--dts 0.0001,0.0002,0.0005,0.001,0.002,0.005,0.01]

The paper's thermalised fluids are not available: dem_inputs.fig3_state gives seeded stand-ins (units sigma = epsilon =
m = 1), thermalised here with --equil time units of NVE in a DEM_F64 context; every run starts from that same state.
A DEM_F32 context evaluates forces in FP32 and integrates the state in double (R15b).  Runs on the CUDA
library only.  Prints one markdown table.
"""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import dem_inputs as di  # noqa: E402

SKIN = 0.4
RECORDS = 200


def thermalise(pkg, st, time_units, dt=5e-3):
    import torch

    dem, t = pkg.from_state(st, "f64")
    f = torch.empty((st["N"], 4), dtype=torch.float64, device="cuda")
    dem.step(t["pos"], t["quat"], t["vel"], t["angmom"], t["shape_id"], st["box"], dt, int(round(time_units / dt)), SKIN, f)
    out = dict(st)
    for k in ("pos", "quat", "vel", "angmom"):
        out[k] = t[k].cpu().numpy()
    dem.close()
    return out


def sigma_e(pkg, st, precision, dt, duration, records=RECORDS):
    """sigma(E/N) over `duration`, E recorded `records` times at equal intervals; also mean E/N and U/N."""
    import torch

    dem, t = pkg.from_state(st, precision)
    f = torch.empty((st["N"], 4), dtype=dem.dtype, device="cuda")
    nsteps = int(round(duration / dt))
    every = max(nsteps // records, 1)
    args = (t["pos"], t["quat"], t["vel"], t["angmom"], t["shape_id"], st["box"], dt)
    dem.step(*args, 0, SKIN, f)
    e = [dem.energy(t["quat"], t["vel"], t["angmom"], t["shape_id"], f)]
    for _ in range(nsteps // every):
        dem.step(*args, every, SKIN, f)
        e.append(dem.energy(t["quat"], t["vel"], t["angmom"], t["shape_id"], f))
    dem.close()
    e = np.array(e) / st["N"]
    return float(e.sum(1).std()), float(e.sum(1).mean()), float(e[:, 0].mean())


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--duration", type=float, default=10.0)
    ap.add_argument("--equil", type=float, default=20.0)
    ap.add_argument("--dts", default="0.0001,0.0002,0.0005,0.001,0.002,0.005,0.01")
    a = ap.parse_args(argv)
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("fig3 needs a CUDA device: the product has no CPU path")
    import paper_1607_02427_b200 as pkg

    dts = [float(x) for x in a.dts.split(",")]
    print("| system | dt / tau | sigma(E/N), DEM_F32 | sigma(E/N), DEM_F64 | <E/N> | <U/N> |")
    print("|---|---|---|---|---|---|")
    rows = []
    for kind in ("squares", "tetrahedra"):
        st = thermalise(pkg, di.fig3_state(kind), a.equil)
        for dt in dts:
            s32, _, _ = sigma_e(pkg, st, "f32", dt, a.duration)
            s64, em, um = sigma_e(pkg, st, "f64", dt, a.duration)
            rows.append((kind, dt, s32, s64))
            print("| %s (N = %d) | %g | %.2e | %.2e | %.4f | %.4f |" % (kind, st["N"], dt, s32, s64, em, um), flush=True)
    return rows


if __name__ == "__main__":
    main()
