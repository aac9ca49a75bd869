"""Pins of the oracle's drift step (O1), block list (O4) and output-tile list (O6).
CPU only."""
import math
import os

import numpy as np
import pytest

import gen
import oracle as o

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _segs(**kw):
    base = dict(x0=10.0, y0=10.0, z0=160.0, x1=10.5, y1=10.2, z1=160.0, q=6000.0, t0=0.0)
    base.update(kw)
    return {k: np.array([v], np.float32) for k, v in base.items()}


def test_drift_closed_forms():
    """attachment exp(-t/tau), drift t = z/v, diffusion
    sigma = sqrt(2 D t) (readings G6, G7, G11).  Hand-computed numbers:
    z = 160 mm, v = 1.6 mm/us -> t = 100 us; sigma_T = sqrt(2*1.2e-3*100) = 0.4898979...
    sigma_L = sqrt(2*7.2e-4*100) = 0.3794733... mm -> /v = 0.2371708... us."""
    cfg = gen.make_config(1)
    aug = o.drift(cfg, _segs(t0=3.0))
    assert abs(aug["p0"][0, 2] - 103.0) < 1e-12 and abs(aug["p1"][0, 2] - 103.0) < 1e-12
    assert abs(aug["tm"][0] - 100.0) < 1e-12                    # excludes t0
    assert abs(aug["sig"][0, 0] - 0.4898979485566356) < 1e-12
    assert abs(aug["sig"][0, 1] - 0.4898979485566356) < 1e-12
    assert abs(aug["sig"][0, 2] - 0.2371708245126284) < 1e-12
    assert abs(aug["Qp"][0] - 6000.0 * math.exp(-100.0 / 2200.0)) < 1e-9
    assert abs(aug["Qp"][0] / 6000.0 - 0.955563) < 1e-6               # 1 - x + x^2/2 - x^3/6, x = 1/22
    # minimum diffusion scale (reading G8) at z -> 0
    aug0 = o.drift(cfg, _segs(z0=0.0, z1=0.01))
    assert aug0["sig"][0, 0] == cfg.sigma_min_xy_mm and aug0["sig"][0, 2] == cfg.sigma_min_t_us


def test_point_flag_threshold():
    """point-like iff every |d_a| < 0.1 sigma_a (strict, reading G10)."""
    cfg = gen.make_config(1)
    s = 0.4898979485566356
    assert o.drift(cfg, _segs(x1=10.0 + 0.09 * s, y1=10.0))["flag"][0] == 1
    assert o.drift(cfg, _segs(x1=10.0 + 0.11 * s, y1=10.0))["flag"][0] == 0
    # the time axis counts too: dz = 0.1 mm -> dt = 0.0625 us > 0.1 * 0.237
    assert o.drift(cfg, _segs(x1=10.0, y1=10.0, z1=160.1))["flag"][0] == 0


def test_bbox_brute_force():
    """bbox = cuboids meeting [min end - nsigma sigma, max end + nsigma sigma] (G9):
    checked by testing every cuboid interval against the continuous box."""
    cfg, segs = gen.make_segments(1)
    aug = o.drift(cfg, segs)
    g = o.grid_of(cfg)
    for s in range(0, 300, 17):
        for a in range(3):
            lo_c = min(aug["p0"][s, a], aug["p1"][s, a]) - cfg.nsigma * aug["sig"][s, a]
            hi_c = max(aug["p0"][s, a], aug["p1"][s, a]) + cfg.nsigma * aug["sig"][s, a]
            idx = np.arange(aug["lo"][s, a] - 3, aug["hi"][s, a] + 4)
            left = g.org[a] + idx * g.h[a]
            inside = (left + g.h[a] > lo_c) & (left <= hi_c)
            got = (idx >= aug["lo"][s, a]) & (idx <= aug["hi"][s, a])
            # cuboid edges that coincide with the box edge to rounding may differ
            edge = (np.abs(left + g.h[a] - lo_c) < 1e-9) | (np.abs(left - hi_c) < 1e-9)
            assert ((inside == got) | edge).all()


def test_blocks_cover_all_charge_and_reassemble():
    """O4 by brute force: scatter Eq. (9) of every segment into ALL blocks of a small
    plane; every non-zero must lie in a block of the footprint list, and the list is
    sorted and unique."""
    cfg, segs = gen.make_segments(1)
    cfg = cfg.with_(nticks=512)
    segs = {k: v[:40] for k, v in segs.items()}
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    assert (np.diff(keys) > 0).all()
    g = o.grid_of(cfg)
    allkeys = np.arange(g.NB[0] * g.NB[1] * g.NB[2], dtype=np.int64)
    full = o.effq(cfg, aug, allkeys)
    occupied = np.flatnonzero(np.abs(full).reshape(len(allkeys), -1).sum(1) > 0)
    assert np.isin(occupied, keys).all()
    assert len(occupied) > 0.5 * len(keys)           # the footprint list is not wildly loose
    sub = o.effq(cfg, aug, keys)
    np.testing.assert_allclose(sub, full[keys], rtol=1e-12, atol=0)   # omp summation order
    # key layout (reading G16): slab-major, then x, then y
    bx, by, bt = o.key_to_bxyz(g, keys)
    np.testing.assert_array_equal(keys, (bt * g.NB[0] + bx) * g.NB[1] + by)


def test_block_pairs_match_python_loop():
    cfg, segs = gen.make_segments(1)
    segs = {k: v[:25] for k, v in segs.items()}
    aug = o.drift(cfg, segs)
    g = o.grid_of(cfg)
    seg, keys, cnt = o.block_pairs(cfg, aug)
    ref = []
    e = 1
    for s in range(25):
        lo = np.maximum(aug["lo"][s] - e, 0)
        hi = np.minimum(aug["hi"][s] + e, np.array(g.NG) - 1)
        if (lo > hi).any():
            continue
        for bt in range(lo[2] // g.B[2], hi[2] // g.B[2] + 1):
            for bx in range(lo[0] // g.B[0], hi[0] // g.B[0] + 1):
                for by in range(lo[1] // g.B[1], hi[1] // g.B[1] + 1):
                    ref.append((s, (bt * g.NB[0] + bx) * g.NB[1] + by))
    assert list(zip(seg.tolist(), keys.tolist())) == ref


def test_out_tiles_cover_all_current():
    """O6 by brute force: every (pixel, tick) with non-zero current of a direct
    convolution lies in a listed tile."""
    cfg, segs = gen.make_segments(1)
    cfg = cfg.with_(nticks=512, npix_x=16, npix_y=16, resp_nticks=40)
    segs = {k: v[:12] for k, v in segs.items()}
    # move the 12 segments into the small plane
    for k in ("x0", "x1"):
        segs[k] = (segs[k] - segs["x0"][0] + 30.0).astype(np.float32)
    for k in ("y0", "y1"):
        segs[k] = (segs[k] - segs["y0"][0] + 30.0).astype(np.float32)
    R = gen.make_random_response(cfg, 5)
    res = o.simulate(cfg, segs, R)
    tiles = res["tiles"]
    assert (np.diff(tiles) > 0).all()
    g = o.grid_of(cfg)
    Tt = g.B[2]
    nz = np.argwhere(res["wave"] != 0.0)
    px, py = nz[:, 0] // cfg.npix_y, nz[:, 0] % cfg.npix_y
    tk = ((nz[:, 1] // Tt) * cfg.npix_x + px) * cfg.npix_y + py
    assert len(nz) > 0 and np.isin(np.unique(tk), tiles).all()


def test_paper_padding_example():
    """tests/golden/paper_padding.txt: linear-convolution sizes."""
    for line in open(os.path.join(GOLD, "paper_padding.txt")):
        f = line.split("#")[0].split()
        if len(f) == 4:
            n_in, n_resp, exact, pow2 = map(int, f)
            assert n_in + n_resp - 1 == exact
            n = 1
            while n < exact:
                n *= 2
            assert n == pow2


@pytest.mark.parametrize("tr", [65, 66])
def test_out_tiles_exact_by_brute_force(tr):
    """O6 pinned to equality: blocks filled with ones, a response of ones on every offset, phase
    and tick, direct sum of Eq. (12).  Everything is positive, so the support of
    the current IS the output footprint of the blocks, and its tiles must EQUAL the list -- no
    tile too few and none too many.  Bt = 64: with Tr = 65 a block's last output tick
    Bt bt + Bt + Tr - 2 is the last tick of tile bt + 1, with Tr = 66 the first tick of tile
    bt + 2; a footprint one tick too long or too short fails one of the two.  The blocks include
    ones that straddle two pixels (8 fine points per block, 10 per pixel), ones at the plane's
    rim and one whose output runs past the readout window."""
    cfg = gen.make_config(1).with_(npix_x=12, npix_y=10, nticks=400, resp_nticks=tr, resp_half=1)
    g = o.grid_of(cfg)
    assert g.B == (8, 8, 64) and cfg.sub == 10
    blocks = [(0, 0, 0), (1, 5, 0), (6, 3, 1), (14, 12, 2), (7, 7, 3), (3, 9, 5), (9, 2, 6)]
    keys = np.array(sorted((bt * g.NB[0] + bx) * g.NB[1] + by for bx, by, bt in blocks), dtype=np.int64)
    payload = np.ones((len(keys),) + tuple(g.B))
    K = 2 * cfg.resp_half + 1
    R = np.ones((cfg.sub, cfg.sub, K, K, tr), dtype=np.float32)
    pix = np.arange(cfg.npix_x * cfg.npix_y, dtype=np.int64)
    wave = o.conv_direct(cfg, keys, payload, R, pix)
    nz = np.argwhere(wave > 0)
    brute = np.unique((nz[:, 1] // g.B[2]) * (cfg.npix_x * cfg.npix_y) + nz[:, 0])
    np.testing.assert_array_equal(o.out_tiles(cfg, keys), brute)
    # the support itself, per block, is the stated box (pixels and ticks), not just its tiles
    bx, by, bt = o.key_to_bxyz(g, keys[:1])
    on = np.zeros_like(wave, dtype=bool)
    for x, y, t in blocks:
        px0, px1 = max(8 * x // 10 - 1, 0), min((8 * x + 7) // 10 + 1, cfg.npix_x - 1)
        py0, py1 = max(8 * y // 10 - 1, 0), min((8 * y + 7) // 10 + 1, cfg.npix_y - 1)
        t1 = min(64 * t + 64 + tr - 2, cfg.nticks - 1)
        for px in range(px0, px1 + 1):
            on[px * cfg.npix_y + py0: px * cfg.npix_y + py1 + 1, 64 * t: t1 + 1] = True
    np.testing.assert_array_equal(wave > 0, on)
