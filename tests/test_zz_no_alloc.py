"""dem_energy_static (include/dem.h): the entry point that allocates nothing -- its scratch is a fixed device array inside
the library -- against dem_energy, the existing path, on two calls in a row that share that array.  Collected last on
purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import dem_inputs as di

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: the product has no CPU path")
    import paper_1607_02427_b200 as p

    p.lib()
    return p


@pytest.mark.parametrize("precision,kind,cells", [("f32", "mixed", 10), ("f64", "squares", 24)])
def test_energy_static_matches_dem_energy_on_two_calls_in_a_row(pkg, precision, kind, cells):
    import torch

    st = di.dense_state(kind, cells)
    n = st["N"]
    dem, t = pkg.from_state(st, precision)
    dem.build_neighbors(t["pos"], t["shape_id"], st["box"], st["r_cut"])
    f, _, _ = dem.compute(t["pos"], t["quat"], t["shape_id"], virial=False)
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    # first call: the whole state (several blocks and a ragged tail)
    want1 = dem.energy(t["quat"], t["vel"], t["angmom"], t["shape_id"], f)
    dem.energy_static(t["quat"], t["vel"], t["angmom"], t["shape_id"], f, out)
    got1 = out.cpu().numpy()
    # second call, straight after, on fewer particles with other velocities: it uses fewer blocks, so the array still
    # holds the first call's sums beyond them, which must not be read
    m = n // 3 + 1
    sub = {k: t[k][:m].contiguous() for k in ("quat", "vel", "angmom", "shape_id")}
    sub["vel"] = sub["vel"] * 1.5
    fs = f[:m].contiguous()
    out2 = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    dem.energy_static(sub["quat"], sub["vel"], sub["angmom"], sub["shape_id"], fs, out2)
    got2 = out2.cpu().numpy()
    want2 = dem.energy(sub["quat"], sub["vel"], sub["angmom"], sub["shape_id"], fs)
    # and the first inputs once more: the result is that of the first call, bit for bit (fixed summation order)
    dem.energy_static(t["quat"], t["vel"], t["angmom"], t["shape_id"], f, out)
    got3 = out.cpu().numpy()
    dem.close()
    assert np.all(np.isfinite(got1)) and np.all(np.isfinite(got2))
    assert abs(want1[0]) > 0 and want1[1] > 0 and want1[2] > 0          # the state interacts, moves and spins
    # the two paths add the same per-particle doubles in different orders: relative 1e-12 of each sum's magnitude
    for got, want in ((got1, want1), (got2, want2)):
        assert np.all(np.abs(got - want) <= 1e-12 * np.maximum(np.abs(want), 1.0)), (got, want)
    assert abs(want2[1] - want1[1]) > 1e-3 * want1[1]                    # the second call really was another problem
    assert np.array_equal(got3, got1)


def test_energy_static_rejects_sizes_beyond_its_scratch(pkg):
    import torch

    st = di.dense_state("squares", 8)
    dem, t = pkg.from_state(st, "f32")
    n = (1 << 20) + 1                                                    # DEM_ENERGY_STATIC_MAX_N + 1
    z4 = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
    sid = torch.zeros((n,), dtype=torch.int32, device="cuda")
    out = torch.zeros((3,), dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.DemError) as e:
        dem.energy_static(z4, z4, z4, sid, z4, out)
    assert "DEM_ENERGY_STATIC_MAX_N" in str(e.value)
    # the largest size it accepts runs (zero state: all three sums are zero)
    out.fill_(float("nan"))
    dem.energy_static(z4[:-1], z4[:-1], z4[:-1], sid[:-1], z4[:-1], out)
    assert np.array_equal(out.cpu().numpy(), np.zeros(3))
    dem.close()
