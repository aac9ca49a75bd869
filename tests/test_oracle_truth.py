"""Pins of the oracle's truth record (DESIGN.md
reading G24): it partitions each segment's charge, and it adds up to what the pixels collect."""
import numpy as np

import gen
import oracle as o


def _case():
    """30 consecutive segments of a config-2 track that stay 7 pixels clear of the plane's rim
    and inside the time window (so that nothing is clipped)."""
    cfg, segs = gen.make_segments(2)
    m = 7 * cfg.pitch_mm
    ok = np.ones(len(segs["q"]), bool)
    for k, n in (("x0", cfg.npix_x), ("x1", cfg.npix_x), ("y0", cfg.npix_y), ("y1", cfg.npix_y)):
        ok &= (segs[k] > m) & (segs[k] < n * cfg.pitch_mm - m)
    t = (np.maximum(segs["z0"], segs["z1"]) / cfg.v_mm_us - cfg.t_origin_us) / cfg.tick_us
    ok &= t < cfg.nticks - cfg.resp_nticks - 2 * cfg.block[2]
    runs = np.flatnonzero(np.convolve(ok.astype(int), np.ones(30, int), "valid") == 30)
    assert len(runs) > 0
    i0 = int(runs[0])
    segs = {k: v[i0:i0 + 30] for k, v in segs.items()}
    return cfg, segs, o.drift(cfg, segs)


def test_records_partition_the_segment_charge():
    cfg, segs, aug = _case()
    rs, rk, rq = o.truth_record(cfg, aug)
    tot = np.bincount(rs, weights=rq, minlength=len(aug["Qp"]))
    keys = o.blocks(cfg, aug)
    per_seg = np.array([o.effq(cfg, aug, keys, [s]).sum() for s in range(len(aug["Qp"]))])
    assert np.allclose(tot, per_seg, rtol=1e-12)              # every grid point belongs to exactly one entry
    inside = (aug["lo"].min(1) >= 1) & (aug["hi"][:, 0] < cfg.npix_x * cfg.sub - 1) & \
             (aug["hi"][:, 1] < cfg.npix_y * cfg.sub - 1) & (aug["hi"][:, 2] < cfg.nticks - 1)
    assert inside.any()
    assert np.allclose(tot[inside], aug["Qp"][inside], rtol=3e-4)      # = Q exp(-t/tau) up to the 4-sigma box
    # keys: sorted within a segment, inside the plane and the window
    for s in np.unique(rs):
        k = rk[rs == s]
        assert np.all(np.diff(k) > 0)
    npix = cfg.npix_x * cfg.npix_y
    assert rk.min() >= 0 and (rk // npix).max() < -(-cfg.nticks // cfg.block[2])


def test_records_add_up_to_the_collected_charge():
    """The synthetic response integrates to 1 on the collecting pixel and to 0 elsewhere
    (reading G18), so the time integral of a pixel's waveform is the charge the truth
    record books on that pixel."""
    cfg, segs, aug = _case()
    R = gen.make_response(cfg, 2002)
    rs, rk, rq = o.truth_record(cfg, aug)
    npix = cfg.npix_x * cfg.npix_y
    per_pixel = np.bincount(rk % npix, weights=rq, minlength=npix)
    pix = np.flatnonzero(per_pixel > 0.05 * per_pixel.max())
    pix = pix[(pix // cfg.npix_y > 5) & (pix // cfg.npix_y < cfg.npix_x - 6) &
              (pix % cfg.npix_y > 5) & (pix % cfg.npix_y < cfg.npix_y - 6)][:6]
    assert len(pix) >= 2
    sim = o.simulate(cfg, segs, R, pix=pix, fft=True)
    last = rk // npix
    assert (last.max() + 1) * cfg.block[2] + cfg.resp_nticks <= cfg.nticks      # nothing truncated in time
    assert np.allclose(sim["wave"].sum(1), per_pixel[pix], rtol=1e-6)


def test_record_keys_by_dense_box_sums_and_arrival_tick():
    """The (pixel, time tile) index of every entry, pinned twice without truth_record's own
    per-block bookkeeping: (1) the segment's effective charge scattered onto the dense fine
    grid and summed over S x S x Bt boxes by a reshape gives the same keys and the same charges;
    (2) the tile that books most of a segment's charge is the one holding its arrival tick
    (z / v - t_origin) / tick (reading G11) whenever the charge cloud lies well
    inside that tile."""
    cfg, segs = gen.make_segments(1)
    cfg = cfg.with_(npix_x=16, npix_y=16, nticks=512)
    segs = {k: v[40:64].copy() for k, v in segs.items()}
    for a in ("x", "y"):                               # move the piece of track into the small plane
        sh = 35.0 - segs[a + "0"][0]
        segs[a + "0"] = (segs[a + "0"] + sh).astype(np.float32)
        segs[a + "1"] = (segs[a + "1"] + sh).astype(np.float32)
    zs = 120.0 - segs["z0"][0]
    segs["z0"] = (segs["z0"] + zs).astype(np.float32)
    segs["z1"] = (segs["z1"] + zs).astype(np.float32)
    cfg = cfg.with_(t_origin_us=float(segs["z0"].min() / cfg.v_mm_us - 8.0))
    aug = o.drift(cfg, segs)
    rs, rk, rq = o.truth_record(cfg, aug)
    g = o.grid_of(cfg)
    S, Bt = cfg.sub, cfg.block[2]
    npix = cfg.npix_x * cfg.npix_y
    ntb = g.NG[2] // Bt
    keys = o.blocks(cfg, aug)
    checked = dominant = 0
    for s in range(len(aug["Qp"])):
        dense = o.payload_to_dense(cfg, keys, o.effq(cfg, aug, keys, [s]))
        box = dense.reshape(cfg.npix_x, S, cfg.npix_y, S, ntb, Bt).sum((1, 3, 5))      # [px][py][tb]
        ref = {(tb * cfg.npix_x + px) * cfg.npix_y + py: box[px, py, tb] for px, py, tb in np.argwhere(box != 0)}
        got = dict(zip(rk[rs == s].tolist(), rq[rs == s].tolist()))
        # an entry may be an exact zero (a footprint cell the 4-sigma box reaches with underflow); not vice versa
        assert set(ref) <= set(got)
        for k, v in got.items():
            assert abs(v - ref.get(k, 0.0)) <= 1e-12 * max(abs(v), 1e-300) + 1e-300
        checked += len(ref)
        # (2) arrival tick of the segment's midpoint, cloud (4 sigma + half length) inside one tile
        tick_mid = (0.5 * (aug["p0"][s, 2] + aug["p1"][s, 2]) - cfg.t_origin_us) / cfg.tick_us
        half = 0.5 * abs(aug["p1"][s, 2] - aug["p0"][s, 2]) / cfg.tick_us + cfg.nsigma * aug["sig"][s, 2] / cfg.tick_us
        tb = int(tick_mid // Bt)
        if tick_mid - half > tb * Bt + 1 and tick_mid + half < (tb + 1) * Bt - 1:
            per_tb = np.bincount(rk[rs == s] // npix, weights=rq[rs == s], minlength=ntb)
            assert per_tb.argmax() == tb and per_tb[tb] >= (1 - 1e-3) * per_tb.sum()
            dominant += 1
    assert checked > 50 and dominant >= 5
