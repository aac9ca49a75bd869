"""Pins of the oracle's G4Step preprocessing (
DESIGN.md readings G21, G22): hand-worked recombination values, conservation laws of the
splitting, limits."""
import os

import numpy as np

import gen
import oracle as o

HERE = os.path.dirname(os.path.abspath(__file__))


def test_recombination_hand_values():
    for line in open(os.path.join(HERE, "golden", "recombination.txt")):
        if line.startswith("#") or not line.strip():
            continue
        model, dedx, R = line.split()
        par = dict(gen.STEP_PARAMS, recomb_model=int(model))
        assert abs(float(o.recombination(par, [float(dedx)])[0]) - float(R)) < 2e-6


def test_recombination_shape():
    x = np.linspace(2.0, 40.0, 200)         # from about minimum ionising up (the box model's domain)
    for model in (0, 1):
        R = o.recombination(dict(gen.STEP_PARAMS, recomb_model=model), x)
        assert np.all(R > 0) and np.all(R < 1)
        assert np.all(np.diff(R) < 0)                  # more ionisation density, more recombination
    # Birks at zero density of ionisation: nothing recombines beyond the constant A
    assert o.recombination(dict(gen.STEP_PARAMS, recomb_model=0), [0.0])[0] == gen.STEP_PARAMS["birks_A"]
    # the box model is clipped where its logarithm turns negative
    assert o.recombination(dict(gen.STEP_PARAMS, recomb_model=1), [1e-3])[0] == 0.0


def test_split_conserves_and_bounds():
    steps = gen.make_steps(11)
    par = gen.STEP_PARAMS
    r = o.split_steps(par, steps)
    s, parent, count = r["segs"], r["parent"], r["count"]
    p0 = np.stack([s["x0"], s["y0"], s["z0"]], 1).astype(np.float64)
    p1 = np.stack([s["x1"], s["y1"], s["z1"]], 1).astype(np.float64)
    ln = np.linalg.norm(p1 - p0, axis=1)
    assert ln.max() <= par["max_len_mm"] * (1 + 1e-6)                     # every piece within the threshold
    L = np.linalg.norm(np.stack([steps["x1"] - steps["x0"], steps["y1"] - steps["y0"],
                                 steps["z1"] - steps["z0"]], 1).astype(np.float64), axis=1)
    assert np.array_equal(count, np.maximum(np.ceil(L / par["max_len_mm"]), 1).astype(np.int32))
    assert count.sum() == len(parent) and np.all(np.diff(parent) >= 0)
    short = L <= par["max_len_mm"]
    assert np.all(count[short] == 1)                                      # short steps unchanged
    i = np.flatnonzero(short)[0]
    j = np.flatnonzero(parent == i)[0]
    assert s["x0"][j] == steps["x0"][i] and s["z1"][j] == steps["z1"][i]
    # pieces of a step: contiguous, equal length, equal charge (same dE/dx), lengths and charge add up
    first = np.cumsum(count) - count
    qsum = np.bincount(parent, weights=s["q"].astype(np.float64))
    lsum = np.bincount(parent, weights=ln)
    dedx = np.where(L > 0, steps["dE"].astype(np.float64) / L * 10.0, 0.0)
    ne = steps["dE"].astype(np.float64) * 1e6 / par["w_ion_ev"] * o.recombination(par, dedx)
    assert np.allclose(qsum, ne, rtol=2e-6)
    assert np.allclose(lsum, L, rtol=1e-5, atol=1e-4)
    k = int(np.argmax(count))
    a, b = first[k], first[k] + count[k]
    assert np.allclose(p1[a:b - 1], p0[a + 1:b], atol=2e-4)               # fp32 rounding of the joints
    assert np.ptp(ln[a:b]) < 1e-3 and np.ptp(s["q"][a:b]) == 0.0
    assert np.all(s["t0"][a:b] == steps["t0"][k])


def test_split_threshold_edge():
    par = dict(gen.STEP_PARAMS, max_len_mm=5.0)
    st = {k: np.zeros(3, np.float32) for k in gen.STEP_FIELDS}
    st["x1"][:] = [5.0, 5.0000005, 10.000001]          # exactly the threshold, just above, just above 2x
    st["dE"][:] = 1.0
    r = o.split_steps(par, st)
    assert list(r["count"]) == [1, 2, 3]
