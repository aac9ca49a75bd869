"""Pins of the oracle's trigger-reset readout (
DESIGN.md reading G23): closed forms for constant currents and impulses, charge bookkeeping."""
import numpy as np

import oracle as o

PAR = dict(threshold_e=3000.0, n_integ=16, n_reset=8, max_hits=8, adc_lsb_e=0.0)


def test_constant_current_is_periodic():
    """I0 per tick: fires when (k+1) I0 >= T, i.e. k = ceil(T/I0) - 1; record n_integ ticks later
    holds (k + 1 + n_integ) I0; after n_reset dead ticks the cycle repeats from zero."""
    I0, n = 250.0, 400
    nh, tick, adc = o.readout(PAR, np.full((1, n), I0, np.float32))
    k = int(np.ceil(PAR["threshold_e"] / I0)) - 1
    period = k + PAR["n_integ"] + PAR["n_reset"] + 1
    first = k + PAR["n_integ"]
    expect = [first + j * period for j in range(PAR["max_hits"]) if first + j * period < n]
    assert nh[0] == len(expect) and list(tick[0, :nh[0]]) == expect
    assert np.all(adc[0, :nh[0]] == (k + 1 + PAR["n_integ"]) * I0)


def test_impulse_and_subthreshold():
    w = np.zeros((3, 200), np.float32)
    w[0, 50] = 6000.0                       # one hit, n_integ later, full charge
    w[1, :] = 10.0                          # 2000 e in total: never fires
    w[2, 40] = 6000.0; w[2, 40 + 16 + 3] = 5000.0     # second pulse inside the dead time: lost
    nh, tick, adc = o.readout(PAR, w)
    assert nh[0] == 1 and tick[0, 0] == 66 and adc[0, 0] == 6000.0 and tick[0, 1] == -1
    assert nh[1] == 0
    assert nh[2] == 1 and adc[2, 0] == 6000.0
    # hit whose sampling time falls beyond the window is not recorded
    w2 = np.zeros((1, 60), np.float32); w2[0, 50] = 6000.0
    assert o.readout(PAR, w2)[0][0] == 0


def test_charge_bookkeeping():
    """sum of records + charge of the dead ticks + what is left on the channel = total charge."""
    rng = np.random.default_rng(3)
    w = (rng.random((6, 600)) < 0.05) * rng.uniform(500, 4000, (6, 600))
    w = w.astype(np.float32)
    par = dict(PAR, max_hits=64)
    nh, tick, adc = o.readout(par, w)
    for p in range(6):
        dead = np.zeros(600, bool)
        for h in range(nh[p]):
            dead[tick[p, h] + 1: tick[p, h] + 1 + par["n_reset"]] = True
        last = tick[p, nh[p] - 1] + par["n_reset"] + 1 if nh[p] else 0
        left = w[p, last:].sum(dtype=np.float64)
        total = w[p].sum(dtype=np.float64)
        assert abs(adc[p, :nh[p]].sum(dtype=np.float64) + w[p, dead].sum(dtype=np.float64) + left - total) < 1e-2
    assert nh.max() > 1


def test_noise_terms_and_quantisation():
    w = np.zeros((1, 300), np.float32); w[0, 20:60] = 200.0; w[0, 150:190] = 200.0
    noise = np.zeros((1, 8, 3), np.float32)
    noise[0, 0] = (-1000.0, 123.0, 400.0)      # lower threshold fires 5 ticks earlier; adc offset; baseline
    nh0, t0, a0 = o.readout(PAR, w)
    nh1, t1, a1 = o.readout(PAR, w, noise)
    assert t0[0, 0] - t1[0, 0] == 5
    assert a1[0, 0] == np.float32((t1[0, 0] - 20 + 1) * 200.0 + 123.0)
    # second record, by hand.  Without noise: dead ticks 51..58, tick 59 leaves 200 e on the
    # channel, 200 + 14*200 >= 3000 at tick 163, record at 179 with 200 + 30*200.  With the
    # draws: dead 46..53, baseline 400 + ticks 54..59 = 1600, 1600 + 7*200 >= 3000 at tick 156,
    # record at 172 with 1600 + 23*200.
    assert (t0[0, 1], t1[0, 1]) == (179, 172)
    assert a0[0, 1] == 200.0 + 30 * 200.0 and a1[0, 1] == 1600.0 + 23 * 200.0
    q = o.readout(dict(PAR, adc_lsb_e=250.0), w)[2]
    assert np.all(np.mod(q[0, :nh0[0]], 250.0) == 0)
