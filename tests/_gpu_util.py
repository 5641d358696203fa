"""Helpers for the GPU parity tests: run the CUDA path through the C ABI binding and compare with the oracle."""
import numpy as np

TOL = {"f32": 1e-4, "f64": 1e-10}  # north_star: relative to the system's max |F| (floored by eps/sigma, reading R19)


def round_state(st, precision):
    """The oracle must see the same stored values as the GPU: FP32 runs promote the rounded floats to double."""
    st = dict(st)
    if precision == "f32":
        for k in ("pos", "quat", "vel", "angmom"):
            st[k] = st[k].astype(np.float32).astype(np.float64)
    return st


def scales(st, of, ot):
    sig = min(2 * s["rounding"] for s in st["shapes"])
    eps = st.get("epsilon", 1.0)
    return max(np.abs(of[:, :3]).max(), eps / sig), max(np.abs(ot[:, :3]).max(), eps), max(np.abs(of[:, 3]).max(), eps)


def gpu_compute(st, precision, slices=0, r_cut=None, virial=True, kernel=None, cull=None):
    import paper_1607_02427_b200 as pkg

    dem, t = pkg.from_state(st, precision)
    if slices:
        dem.set_slices(slices)
    if kernel is not None:
        dem.set_pair_kernel(kernel)
    if cull is not None:
        dem.set_culling(cull)
    dem.build_neighbors(t["pos"], t["shape_id"], st["box"], st["r_cut"] if r_cut is None else r_cut)
    f, tq, w = dem.compute(t["pos"], t["quat"], t["shape_id"], virial=virial)
    out = (f.cpu().numpy().astype(np.float64), tq.cpu().numpy().astype(np.float64),
           None if w is None else w.cpu().numpy().astype(np.float64), dem.get_counters())
    dem.close()
    return out


def assert_parity(st, precision, oracle, slices=0, subset=None, r_cut=None, tol=None, kernel=None, cull=None, wlever=None):
    """Element-by-element comparison of force, torque, energy, virial and of the term counters.  wlever: a length; the
    virial W = -1/2 d x F is then compared relative to at least wlever x (force scale) -- for states whose centre
    separations |d| are much longer than the contact gaps, where |d| times the force tolerance exceeds max |W|."""
    st = round_state(st, precision)
    f, tq, w, cnt = gpu_compute(st, precision, slices, r_cut, kernel=kernel, cull=cull)
    of, ot, ow, ocnt = oracle.compute(st, subset=subset)
    if subset is not None:
        f, tq, w = f[subset], tq[subset], w[subset]
    fs, ts, us = scales(st, of, ot)
    tol = TOL[precision] if tol is None else tol
    ef = np.abs(f[:, :3] - of[:, :3]).max() / fs
    et = np.abs(tq[:, :3] - ot[:, :3]).max() / ts
    eu = np.abs(f[:, 3] - of[:, 3]).max() / us
    ws = max(np.abs(ow).max(), 1.0, (wlever or 0.0) * fs)
    ew = np.abs(w - ow).max() / ws
    assert ef < tol, "force error %.3e (scale %.3g)" % (ef, fs)
    assert et < tol, "torque error %.3e (scale %.3g)" % (et, ts)
    assert eu < tol, "energy error %.3e" % eu
    assert ew < tol, "virial error %.3e" % ew
    if subset is None:
        # the oracle visits every ordered pair, the GPU every unordered pair once
        assert 2 * cnt["active"] == ocnt[2], (cnt, ocnt)
        assert 2 * cnt["degenerate"] == ocnt[3]
        assert 2 * cnt["parallel"] == ocnt[4], (cnt, ocnt)
    return dict(ef=ef, et=et, eu=eu, ew=ew, counters=cnt, ocounters=ocnt)


def sorted_rows(counts, rows):
    rows = rows.cpu().numpy().astype(np.int64)
    rows = np.where(rows < 0, 2 ** 40, rows)
    return counts.cpu().numpy(), np.sort(rows, axis=1)


def assert_neighbors_exact(st, precision, oracle, r_cut=None, subset=None):
    import paper_1607_02427_b200 as pkg

    st = round_state(st, precision)
    dem, t = pkg.from_state(st, precision)
    rc = st["r_cut"] if r_cut is None else r_cut
    dem.build_neighbors(t["pos"], t["shape_id"], st["box"], rc)
    counts, rows = sorted_rows(*dem.get_neighbors())
    dem.close()
    oc, orows = oracle.neighbors(st, r_cut=rc, subset=subset)
    idx = np.arange(st["N"]) if subset is None else np.asarray(subset)
    assert np.array_equal(counts[idx], oc), "neighbour counts differ"
    for k, i in enumerate(idx):
        assert np.array_equal(rows[i, :oc[k]], orows[k, :oc[k]]), "neighbour row %d differs" % i
    return counts
