"""Parity of the CUDA path (through the C ABI of include/tred.h) with the fp64 oracle,
element by element on the same seeded inputs.  Needs a CUDA device.

Tolerances:
  integers (bbox, flags, block keys, CSR lists, slab/tile keys): bit-exact;
  effective charge (fp32 vs fp64): max|d| <= 2e-5 max|Qeff|, total within 1e-5;
  waveforms: max|d| <= 1e-4 max|signal| (north_star);
  per-pixel integrated charge (north_star: relative 1e-5):
      collecting pixels (|Q_p| >= L1_p / 10, L1_p = sum_t |I_p(t)|: the collection pulse is not
      buried under the bipolar induction of the neighbours, and
      |Q_p| >= 1e-3 max|Q|):  |dQ_p| <= 1e-5 |Q_p|, nothing added;
      every other pixel integrates a bipolar induction pulse to ~0 by cancellation, where a
      relative bound is undefined (reading G17): |dQ_p| <= c 2^-24 L1_p with c from the error
      model of DESIGN.md "Tolerances": c = 4 (fp32 rounding of samples, FFT passes, gather) for
      the fp32 FMA product, plus 3/16 per truncating tensor-core accumulation of the product
      that ran (75 for the tf32 products, 52 for tf32 + 2 x bf16, 39 for the three fp16 products).
"""
import os

import numpy as np
import pytest

import gen
import oracle as o

pytestmark = pytest.mark.gpu

TOL_QEFF = 2e-5
TOL_WAVE = 1e-4
TOL_QPIX = 1e-5
# tensor-core accumulations per output value by spectrum-product kernel (tred_last_mac_mode);
# K2 = 200 reals per row: 25 K-steps of 8 (tf32) or 13 of 16 (bf16 / fp16), three products
N_ACC = {1: 0, 2: 75, 3: 75, 4: 75, 5: 75, 6: 52, 7: 39}


def tol_qpix_l1(mode):
    return (4.0 + 0.1875 * N_ACC[mode]) * 2.0 ** -24


def _torch():
    import torch
    return torch


def _sim(cfg, **kw):
    from paper_2602_12052_b200 import Tred
    return Tred(cfg, **kw)


def _seg_tensor(segs):
    torch = _torch()
    a = np.stack([segs[k] for k in gen.SEG_FIELDS]).astype(np.float32)
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _small(cfg_id):
    """Workloads the oracle finishes in seconds, same recipe as BASELINE configs."""
    if cfg_id == 1:
        return gen.make_segments(1)
    if cfg_id == 2:
        cfg, segs = gen.make_segments(2)
        return cfg, {k: v[:1500] for k, v in segs.items()}
    cfg, segs = gen.make_segments(3, n_vertices=1)
    return cfg, {k: v[:1200] for k, v in segs.items()}


# ------------------------------------------------------------------ S1
@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_drift_bit_exact(cfg_id):
    cfg, segs = gen.make_segments(cfg_id) if cfg_id < 3 else gen.make_segments(3, n_vertices=3)
    aug = o.drift(cfg, segs)
    sim = _sim(cfg)
    augf, augi, npairs = sim.drift(_seg_tensor(segs))
    augi = augi.cpu().numpy()
    augf = augf.cpu().numpy().astype(np.float64)
    np.testing.assert_array_equal(augi[0:3].T, aug["lo"])
    np.testing.assert_array_equal(augi[3:6].T, aug["hi"])
    np.testing.assert_array_equal(augi[6], aug["flag"])
    _, _, cnt = o.block_pairs(cfg, aug)
    np.testing.assert_array_equal(augi[7], cnt)
    assert int(npairs.item()) == int(cnt.sum())
    g = o.grid_of(cfg)
    org, h = np.array(g.org), np.array(g.h)
    p0 = (aug["p0"] - org) / h - aug["lo"]
    p1 = (aug["p1"] - org) / h - aug["lo"]
    np.testing.assert_allclose(augf[0:3].T, p0, atol=4e-6)
    np.testing.assert_allclose(augf[3:6].T, p1, atol=4e-6)
    np.testing.assert_allclose(augf[6:9].T, aug["sig"] / h, rtol=1e-6)
    np.testing.assert_allclose(augf[9], aug["Qp"], rtol=1e-6)


# ------------------------------------------------------------------ S3
def _oracle_csr(cfg, aug):
    seg, keys, _ = o.block_pairs(cfg, aug)
    order = np.argsort(keys, kind="stable")
    ks, ss = keys[order], seg[order]
    uk, first = np.unique(ks, return_index=True)
    off = np.concatenate([first, [len(ks)]])
    return uk, off, ss


@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_blockbin_bit_exact(cfg_id):
    cfg, segs = gen.make_segments(cfg_id) if cfg_id < 3 else gen.make_segments(3, n_vertices=4)
    aug = o.drift(cfg, segs)
    uk, off, ss = _oracle_csr(cfg, aug)
    sim = _sim(cfg)
    augf, augi, npairs = sim.drift(_seg_tensor(segs))
    cap = int(npairs.item())
    keys, blk_off, pair_seg, slab_off, nblocks = sim.blockbin(augi, cap)
    nb = int(nblocks.item())
    assert nb == len(uk)
    np.testing.assert_array_equal(keys[:nb].cpu().numpy(), uk)
    np.testing.assert_array_equal(blk_off[:nb + 1].cpu().numpy(), off)
    np.testing.assert_array_equal(pair_seg[:cap].cpu().numpy(), ss)
    g = o.grid_of(cfg)
    bt = uk // (g.NB[0] * g.NB[1])
    ref_slab = np.searchsorted(bt, np.arange(g.NB[2] + 1), side="left")
    np.testing.assert_array_equal(slab_off.cpu().numpy(), ref_slab)
    np.testing.assert_array_equal(keys[:nb].cpu().numpy(), o.blocks(cfg, aug))


def test_blockbin_capacity_semantics_and_empty():
    cfg, segs = gen.make_segments(1)
    sim = _sim(cfg)
    augf, augi, npairs = sim.drift(_seg_tensor(segs))
    cap = int(npairs.item())
    keys, blk_off, pair_seg, slab_off, nblocks = sim.blockbin(augi, cap, cap_blocks=10)
    full = o.blocks(cfg, o.drift(cfg, segs))
    assert int(nblocks.item()) == len(full)               # required count still reported
    np.testing.assert_array_equal(keys[:10].cpu().numpy(), full[:10])
    # empty input
    torch = _torch()
    empty = torch.empty((8, 0), dtype=torch.float32, device="cuda")
    augf, augi, npairs = sim.drift(empty)
    assert int(npairs.item()) == 0
    keys, blk_off, pair_seg, slab_off, nblocks = sim.blockbin(augi, 0)
    assert int(nblocks.item()) == 0 and int(slab_off.abs().sum().item()) == 0
    out = sim.simulate(empty, sim.prepare_response(torch.zeros(
        (cfg.sub, cfg.sub, 11, 11, cfg.resp_nticks), dtype=torch.float32, device="cuda")))
    assert out["ntiles"] == 0 and out["nblocks"] == 0


# ------------------------------------------------------------------ S2
def _effq_both(cfg, segs, effq_mode=0):
    cfg = cfg.with_(effq_mode=effq_mode)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    ref = o.effq(cfg, aug, keys)
    sim = _sim(cfg)
    augf, augi, npairs = sim.drift(_seg_tensor(segs))
    k, blk_off, pair_seg, slab_off, nblocks = sim.blockbin(augi, int(npairs.item()))
    nb = int(nblocks.item())
    assert nb == len(keys)
    got = sim.effq(nb, k, blk_off, pair_seg, augf, augi)[:nb].cpu().numpy().astype(np.float64)
    return aug, keys, ref, got


@pytest.mark.parametrize("effq_mode", [0, 1])
@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_effq_parity(cfg_id, effq_mode):
    """effq_mode 0: factored line quadrature (default); 1: closed form Eq. (10) per node."""
    cfg, segs = _small(cfg_id)
    aug, keys, ref, got = _effq_both(cfg, segs, effq_mode)
    scale = np.abs(ref).max()
    assert scale > 0
    assert np.abs(got - ref).max() <= TOL_QEFF * scale
    assert abs(got.sum() - ref.sum()) <= 1e-5 * abs(ref.sum())


@pytest.mark.parametrize("effq_mode", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 3, 4])
@pytest.mark.parametrize("block", [(4, 4, 32), (8, 8, 64), (16, 16, 128), (32, 32, 256)])
def test_effq_parity_sweep(n, block, effq_mode):
    """Config 5's representation sweep on a small sample of config-3 inputs."""
    cfg, segs = gen.make_segments(3, n_vertices=1)
    cfg = cfg.with_(gl_n=n, block=block)
    segs = {k: v[:150] for k, v in segs.items()}
    aug, keys, ref, got = _effq_both(cfg, segs, effq_mode)
    assert np.abs(got - ref).max() <= TOL_QEFF * np.abs(ref).max()


def test_effq_factored_long_segments_in_sigmas():
    """The line quadrature picks its order from the segment length in sigmas: 5 mm steps
     at the minimum diffusion scale are ~60 sigma_t long along the drift and
    take several quadrature pieces; a short stub takes the smallest rule."""
    cfg = gen.make_config(1, t_origin_us=0.0, gl_n=3)
    rows = [
        (60.0, 60.0, 2.0, 60.3, 60.2, 7.0, 30000.0, 5.0),          # 5 mm along the drift, sigma_min
        (30.0, 90.0, 1.0, 34.5, 91.0, 1.5, 30000.0, 20.0),         # 4.6 mm across the pixels, sigma_min
        (80.0, 40.0, 100.0, 82.0, 43.0, 103.5, 25000.0, 0.0),      # 5 mm, diffused
        (100.0, 100.0, 120.0, 100.02, 100.3, 120.01, 1800.0, 0.0),  # 0.3 mm stub
    ]
    segs = {k: np.array([r[i] for r in rows], np.float32) for i, k in enumerate(gen.SEG_FIELDS)}
    aug, keys, ref, got = _effq_both(cfg, segs, 0)
    W = np.sqrt((((aug["p1"] - aug["p0"]) / aug["sig"]) ** 2).sum(1))
    assert W.max() > 40 and W.min() < 1.0
    assert np.abs(got - ref).max() <= TOL_QEFF * np.abs(ref).max()
    assert abs(got.sum() - ref.sum()) <= 1e-5 * abs(ref.sum())


def test_effq_modes_agree():
    """The two evaluations of Eq. (10) agree far below the parity tolerance."""
    cfg, segs = _small(2)
    _, _, ref, a = _effq_both(cfg, segs, 0)
    _, _, _, b = _effq_both(cfg, segs, 1)
    assert np.abs(a - b).max() <= 5e-6 * np.abs(ref).max()


@pytest.mark.parametrize("effq_mode", [0, 1])
def test_effq_point_like_and_clipped_segments(effq_mode):
    """Degenerate cases: a point-like stub, a segment straddling the grid edge, one
    wholly outside the grid (no blocks), one at z -> 0 (minimum diffusion scale)."""
    cfg = gen.make_config(1, t_origin_us=0.0)
    rows = [
        (70.0, 70.0, 40.0, 70.01, 70.005, 40.01, 50.0, 0.0),       # point-like
        (-0.3, 30.0, 50.0, 0.6, 30.4, 50.3, 6000.0, 0.0),          # straddles x = 0
        (70.0, 140.5, 60.0, 70.5, 141.2, 60.2, 6000.0, 0.0),       # straddles y max
        (500.0, 500.0, 50.0, 501.0, 500.0, 50.0, 6000.0, 0.0),     # outside: dropped
        (30.0, 30.0, 0.0, 30.5, 30.5, 0.4, 6000.0, 1.0),           # z -> 0, starts at window edge
        (60.0, 60.0, 163.0, 60.5, 60.2, 164.5, 6000.0, 0.0),       # straddles the last tick
    ]
    segs = {k: np.array([r[i] for r in rows], np.float32) for i, k in enumerate(gen.SEG_FIELDS)}
    aug, keys, ref, got = _effq_both(cfg, segs, effq_mode)
    assert aug["flag"][0] == 1 and aug["flag"][1] == 0
    assert np.abs(got - ref).max() <= TOL_QEFF * np.abs(ref).max()


def _effq_with_and_without_tables(cfg, segs, min_blocks=1024):
    """tred_effq twice on the same blocks: with its default workspace (per-segment tables built once)
    and with none (every tile CTA builds the rows it needs)."""
    sim = _sim(cfg)
    augf, augi, npairs = sim.drift(_seg_tensor(segs))
    k, blk_off, pair_seg, slab_off, nblocks = sim.blockbin(augi, int(npairs.item()))
    nb = int(nblocks.item())
    assert nb >= min_blocks, nb                      # below that tred_effq never builds tables
    a = sim.effq(nb, k, blk_off, pair_seg, augf, augi)[:nb].clone()
    b = sim.effq(nb, k, blk_off, pair_seg, augf, augi, work_bytes=0)[:nb]
    _torch().cuda.synchronize()
    return a, b


def test_effq_tables_and_no_tables_give_the_same_bits():
    """The per-segment tables are a cache of what the tile CTAs would compute: same code, same
    bits (tred.h: 'same values, slower'), on a config-3 sample large enough for tables."""
    cfg, segs = gen.make_segments(3, n_vertices=4)
    a, b = _effq_with_and_without_tables(cfg, segs)
    assert float(a.abs().max()) > 0 and bool((a == b).all())


def test_effq_table_offsets_cannot_wrap():
    """Table offsets are int32 sums of table sizes in 16-byte units.  40 000 unsplit segments that
    run ~100 mm along the drift (tables of ~1-2 MB each: hundreds of ticks x hundreds of quadrature
    points) push the sum past 2^31; a wrapped offset must never pass for a valid one (it would
    place a table in front of the workspace).  The library then builds no tables at all, so the
    result must equal the no-table run bit for bit; one segment with a table beyond the per-table
    limit (200 mm) rides along."""
    cfg = gen.make_config(3)
    rng = np.random.default_rng(5)
    n = 40000
    x0 = rng.uniform(20.0, 280.0, n)                 # a 60 x 60 pixel region: ~9 000 blocks, ~1 GB of payload
    y0 = rng.uniform(20.0, 280.0, n)
    z0 = rng.uniform(5.0, 15.0, n)
    dz = rng.uniform(95.0, 105.0, n)
    dz[0] = 200.0
    cols = dict(x0=x0, y0=y0, z0=z0, x1=x0 + rng.uniform(-1.0, 1.0, n), y1=y0 + rng.uniform(-1.0, 1.0, n),
                z1=z0 + dz, q=np.full(n, 5.0e5), t0=np.zeros(n))
    segs = {k: cols[k].astype(np.float32) for k in gen.SEG_FIELDS}
    a, b = _effq_with_and_without_tables(cfg, segs)
    assert float(a.abs().max()) > 0 and bool(_torch().isfinite(a).all()) and bool((a == b).all())
    # the charge is all there: drift attenuation only (lifetime 2200 us, <= 75 us of drift)
    tot = float(a.double().sum())
    assert 0.95 * 5.0e5 * n < tot < 5.0e5 * n * (1 + 1e-6)


# ------------------------------------------------------------------ S4 + S5
def _probe(record: dict):
    """The measured error figures DESIGN.md "Tolerances" quotes: printed (pytest -s), and appended
    as one JSON line to the file TRED_PROBE_OUT names, if set (profiles/r3_error_probe.md gives
    the command that wrote the committed table)."""
    import json
    line = json.dumps(record)
    print("probe:", line)
    path = os.environ.get("TRED_PROBE_OUT")
    if path:
        with open(path, "a") as f:
            f.write(line + "\n")


def _wave_checks(got, ref, mode, tag=None):
    """`mode`: the spectrum-product kernel that ran (Tred.last_mac_mode())."""
    scale = np.abs(ref).max()
    assert scale > 0
    assert np.abs(got - ref).max() <= TOL_WAVE * scale
    qg, qr = got.sum(1), ref.sum(1)
    l1 = np.abs(ref).sum(1)
    dq = np.abs(qg - qr)
    coll = (np.abs(qr) >= 0.1 * l1) & (np.abs(qr) >= 1e-3 * np.abs(qr).max())
    if tag is not None:
        u = 2.0 ** -24
        _probe(dict(tag, mac_mode=int(mode), npix=int(len(l1)), ncollecting=int(coll.sum()),
                    wave_max_err_over_max_signal=float(np.abs(got - ref).max() / scale),
                    dq_over_ulp_l1_collecting=float((dq[coll] / (u * l1[coll])).max()) if coll.any() else None,
                    dq_over_ulp_l1_other=float((dq[~coll & (l1 > 0)] / (u * l1[~coll & (l1 > 0)])).max())
                    if (~coll & (l1 > 0)).any() else None,
                    dq_rel_collecting=float((dq[coll] / np.abs(qr)[coll]).max()) if coll.any() else None,
                    bound_other_ulp_l1=float(tol_qpix_l1(mode) / u)))
    assert (dq[coll] <= TOL_QPIX * np.abs(qr)[coll]).all(), (dq[coll] / np.abs(qr)[coll]).max()
    assert (dq[~coll] <= tol_qpix_l1(mode) * l1[~coll]).all(), (dq[~coll] / l1[~coll]).max() * 2.0 ** 24
    # pixels the oracle leaves exactly empty stay exactly empty
    assert (got[l1 == 0] == 0).all()


def _oracle_charge_pixels(cfg, keys):
    """(slab, pixel) pairs met by an occupied block (O6), as sorted keys."""
    g = o.grid_of(cfg)
    bx, by, bt = o.key_to_bxyz(g, keys)
    S = cfg.sub
    out = set()
    for x, y, t in zip(bx, by, bt):
        for px in range(g.B[0] * x // S, min((g.B[0] * x + g.B[0] - 1) // S, cfg.npix_x - 1) + 1):
            for py in range(g.B[1] * y // S, min((g.B[1] * y + g.B[1] - 1) // S, cfg.npix_y - 1) + 1):
                out.add((int(t) * cfg.npix_x + px) * cfg.npix_y + py)
    return np.array(sorted(out), dtype=np.int64)


@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_plan_tiles_bit_exact(cfg_id):
    torch = _torch()
    cfg, segs = _small(cfg_id)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    sim = _sim(cfg)
    k = torch.from_numpy(keys).cuda()
    npix = cfg.npix_x * cfg.npix_y
    NBt = int(sim.dims.NB[2])
    p = sim.convolve_plan(len(keys), k)
    ref = o.out_tiles(cfg, keys)
    assert int(p["ntiles"].item()) == len(ref)
    np.testing.assert_array_equal(p["tile_keys"][:len(ref)].cpu().numpy(), ref)
    # charge pixels
    cref = _oracle_charge_pixels(cfg, keys)
    assert int(p["ncp"].item()) == len(cref)
    np.testing.assert_array_equal(p["cp_keys"][:len(cref)].cpu().numpy(), cref)
    np.testing.assert_array_equal(p["cp_off"].cpu().numpy(),
                                  np.searchsorted(cref // npix, np.arange(NBt + 1), side="left"))
    # slab-pixel list = the output footprint without the time spread
    spk = p["sp_keys"][:int(p["nsp"].item())].cpu().numpy()
    assert (np.diff(spk) > 0).all()
    g = o.grid_of(cfg)
    bt = keys // (g.NB[0] * g.NB[1])
    assert set(np.unique(spk // npix)) == set(np.unique(bt))
    np.testing.assert_array_equal(p["sp_off"].cpu().numpy(),
                                  np.searchsorted(spk // npix, np.arange(NBt + 1), side="left"))


def _convolve_oracle_charge(sim, cfg, keys, payload32, rhat, pix, work_bytes=None):
    torch = _torch()
    k = torch.from_numpy(keys).cuda()
    p = sim.convolve_plan(len(keys), k)
    ncp, nsp, ntiles = int(p["ncp"].item()), int(p["nsp"].item()), int(p["ntiles"].item())
    sp_data = sim.convolve(len(keys), k, torch.from_numpy(payload32).cuda(), rhat, p, ncp, nsp,
                           p["cp_off"].cpu().numpy(), p["sp_off"].cpu().numpy(), work_bytes=work_bytes)
    tile_data, dense = sim.gather_waveforms(nsp, sp_data, p, ntiles,
                                            torch.from_numpy(pix.astype(np.int32)).cuda())
    return dense.cpu().numpy()


@pytest.mark.parametrize("mac_mode", [1, 0, 2, 3, 4, 5, 6, 7])
@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_convolve_parity_from_oracle_charge(cfg_id, mac_mode):
    """S4+S5 alone: the GPU convolves the ORACLE's effective charge (cast to fp32).
    mac_mode 1: fp32 FMA spectrum product; 0: library default (7 on a B200: three fp16 products);
    the others: include/tred.h.  The kernel that ran is the one asked for (no silent fallback)."""
    torch = _torch()
    cfg, segs = _small(cfg_id)
    cfg = cfg.with_(mac_mode=mac_mode)
    R = gen.make_response(cfg, 2000 + cfg_id)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    payload32 = o.effq(cfg, aug, keys).astype(np.float32)
    rng = np.random.default_rng(cfg_id)
    tiles = o.out_tiles(cfg, keys)
    act = np.unique(tiles % (cfg.npix_x * cfg.npix_y))
    pix = np.sort(rng.choice(act, min(48, len(act)), replace=False))
    ref = o.conv_fft(cfg, keys, payload32.astype(np.float64), R, pix)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    got = _convolve_oracle_charge(sim, cfg, keys, payload32, rhat, pix)
    # mode 4 needs a mirror-symmetric response (this one is) and 100 phases
    assert sim.last_mac_mode() == (7 if mac_mode == 0 else mac_mode)
    _wave_checks(got.astype(np.float64), ref, sim.last_mac_mode(),
                 tag=dict(test="convolve_parity_from_oracle_charge", cfg=cfg_id, requested=mac_mode))


def test_convolve_response_dynamic_range():
    """What the fp16 hi / lo operands of the default product (mac_mode 7) do to a response with a
    wide range between its offsets (include/tred.h, tred_prepare_response): the split uses one
    power-of-two scale per frequency for all offsets, so an offset at rho times that frequency's
    largest entry keeps 22 bits only while rho >= 2^-18; below, its lo part falls into fp16
    subnormals and its own contribution carries a relative error of about 2^-40 / rho.  Here the
    offsets beyond the 3 x 3 centre are scaled down by 1e-5, which with the response's own decay
    puts them at rho = 1e-7 .. 1e-6 of the centre: a pixel that only those offsets reach (induction
    far from all charge) must still come out within 2e-5 of ITS OWN largest sample (2^-40 / rho
    is 1e-6 .. 1e-5), while the fp32 FMA product (mode 1) is held to 5e-6; near pixels keep the
    usual tolerance."""
    torch = _torch()
    cfg = gen.make_config(1, t_origin_us=0.0)
    rows = [(70.0, 70.0, 40.0, 70.9, 70.6, 40.8, 50000.0, 0.0)]          # one short track inside one pixel
    segs = {k: np.array([r[i] for r in rows], np.float32) for i, k in enumerate(gen.SEG_FIELDS)}
    H = cfg.resp_half
    R = gen.make_response(cfg, 2011).astype(np.float64)
    far = np.ones((2 * H + 1, 2 * H + 1))
    far[H - 1:H + 2, H - 1:H + 2] = 0.0
    R *= np.where(far[None, None, :, :, None] > 0, 1.0e-5, 1.0)
    R = np.ascontiguousarray(R, dtype=np.float32)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    payload32 = o.effq(cfg, aug, keys).astype(np.float32)
    # the diffused charge sits on pixels (15..16, 15..16); every `farp` pixel is >= 2 pixels away
    # from all four along at least one axis
    px, py = 15, 15
    assert aug["lo"][0, 0] // cfg.sub == px and aug["hi"][0, 0] // cfg.sub == px + 1
    assert aug["lo"][0, 1] // cfg.sub == py and aug["hi"][0, 1] // cfg.sub == py + 1
    near = [(px, py), (px + 1, py)]
    farp = [(px + 4, py + 3), (px - 3, py + 4), (px + 4, py - 4), (px - 4, py)]
    pix = np.array([a * cfg.npix_y + b for a, b in near + farp])
    order = np.argsort(pix)
    pix = pix[order]
    is_far = np.array([False] * len(near) + [True] * len(farp))[order]
    ref = o.conv_direct(cfg, keys, payload32.astype(np.float64), R, pix)
    own = np.abs(ref).max(1)
    rho = own[is_far] / own[~is_far].max()
    assert rho.max() < 2e-6 and rho.min() > 5e-8, rho
    for mode, tol_far in ((1, 5e-6), (7, 2e-5)):
        sim = _sim(cfg.with_(mac_mode=mode))
        rhat = sim.prepare_response(torch.from_numpy(R).cuda())
        got = _convolve_oracle_charge(sim, cfg, keys, payload32, rhat, pix).astype(np.float64)
        assert sim.last_mac_mode() == mode
        rel = np.abs(got - ref).max(1) / own
        _probe(dict(test="convolve_response_dynamic_range", mac_mode=mode, rho=[float(x) for x in rho],
                    far_err_over_own_max=float(rel[is_far].max()), near_err_over_own_max=float(rel[~is_far].max())))
        assert rel[~is_far].max() <= TOL_WAVE
        assert rel[is_far].max() <= tol_far, (mode, rel[is_far].max())


@pytest.mark.parametrize("block,tr", [((4, 4, 32), 200), ((8, 8, 64), 137), ((16, 16, 128), 400),
                                      ((32, 32, 256), 400), ((8, 8, 32), 225)])
def test_convolve_parity_fft_lengths(block, tr):
    """Config 5's block shapes and odd response lengths: FFT lengths 2^a 3^b with every
    radix mix (432 = 16*27, 256, 576 = 64*9, 768 = 256*3, 256)."""
    torch = _torch()
    cfg, segs = gen.make_segments(1)
    cfg = cfg.with_(block=block, resp_nticks=tr, gl_n=2)
    segs = {k: v[:150] for k, v in segs.items()}
    R = gen.make_random_response(cfg, 5)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    assert len(keys) > 0
    payload32 = o.effq(cfg, aug, keys).astype(np.float32)
    tiles = o.out_tiles(cfg, keys)
    act = np.unique(tiles % (cfg.npix_x * cfg.npix_y))
    pix = act[:: max(1, len(act) // 24)]
    ref = o.conv_fft(cfg, keys, payload32.astype(np.float64), R, pix)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    got = _convolve_oracle_charge(sim, cfg, keys, payload32, rhat, pix).astype(np.float64)
    assert np.abs(got - ref).max() <= TOL_WAVE * np.abs(ref).max()


@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_end_to_end_parity(cfg_id):
    """Whole path, segments in -> waveforms out, against the oracle's direct sum."""
    torch = _torch()
    cfg, segs = _small(cfg_id)
    R = gen.make_response(cfg, 2000 + cfg_id)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    payload = o.effq(cfg, aug, keys)
    tiles = o.out_tiles(cfg, keys)
    act = np.unique(tiles % (cfg.npix_x * cfg.npix_y))
    rng = np.random.default_rng(10 + cfg_id)
    pix = np.sort(rng.choice(act, min(32, len(act)), replace=False))
    ref = o.conv_direct(cfg, keys, payload, R, pix)
    sim = _sim(cfg)
    out = sim.simulate(_seg_tensor(segs), sim.prepare_response(torch.from_numpy(R).cuda()),
                       torch.from_numpy(pix.astype(np.int32)).cuda())
    assert out["nblocks"] == len(keys) and out["ntiles"] == len(tiles)
    np.testing.assert_array_equal(out["tile_keys"].cpu().numpy(), tiles)
    got = out["dense"].cpu().numpy().astype(np.float64)
    _wave_checks(got, ref, sim.last_mac_mode())
    # the sparse tiles hold the same numbers as the dense rows
    tk = out["tile_keys"].cpu().numpy()
    td = out["tile_data"].cpu().numpy()
    npix = cfg.npix_x * cfg.npix_y
    Bt = cfg.block[2]
    for r, p in enumerate(pix[:8]):
        for i in np.flatnonzero(tk % npix == p):
            tb = tk[i] // npix
            n = min(Bt, cfg.nticks - tb * Bt)
            np.testing.assert_array_equal(td[i, :n], out["dense"][r, tb * Bt: tb * Bt + n].cpu().numpy())


def test_convolve_asymmetric_response_and_chunking():
    """An unstructured response pins index order / sign on the GPU too; a small
    workspace forces the slab-group loop, which must give identical bits."""
    torch = _torch()
    cfg, segs = _small(1)
    R = gen.make_random_response(cfg, 77)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    payload = o.effq(cfg, aug, keys)
    pix = np.arange(0, cfg.npix_x * cfg.npix_y, 13)
    ref = o.conv_fft(cfg, keys, payload, R, pix)
    outs = []
    for wb in (None, 1):          # 1 byte -> raised to the minimum (128 charge pixels per chunk)
        sim = _sim(cfg, conv_work_bytes=wb)
        out = sim.simulate(_seg_tensor(segs), sim.prepare_response(torch.from_numpy(R).cuda()),
                           torch.from_numpy(pix.astype(np.int32)).cuda())
        outs.append(out["dense"].cpu().numpy())
    np.testing.assert_array_equal(outs[0], outs[1])
    got = outs[0].astype(np.float64)
    assert np.abs(got - ref).max() <= TOL_WAVE * np.abs(ref).max()
    assert np.abs(got - ref).max() <= 5e-6 * np.abs(ref).max()      # what the path actually gives (2.5e-6)


def test_deterministic_bits():
    """No unordered float atomics anywhere: two runs give identical bits."""
    torch = _torch()
    cfg, segs = _small(2)
    R = gen.make_response(cfg, 2002)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    a = sim.simulate(_seg_tensor(segs), rhat, keep=True)
    b = sim.simulate(_seg_tensor(segs), rhat, keep=True)
    assert torch.equal(a["payload"], b["payload"])
    assert torch.equal(a["tile_data"], b["tile_data"])


@pytest.mark.parametrize("cfg_id", [2, 4])
def test_chunked_equals_single_pass(cfg_id):
    """Config 4's bounded-memory driver: chunks of occupied blocks (ranges of time slabs)
    give the same tile list and bit-identical waveforms as one pass, and parity with the
    oracle on sampled pixels."""
    torch = _torch()
    if cfg_id == 4:
        cfg, segs = gen.make_segments(4, n_vertices=1, n_spills=3)
        segs = {k: v[::40] for k, v in segs.items()}            # keeps the time spread of the pile-up
    else:
        cfg, segs = _small(2)
    R = gen.make_response(cfg, 2000 + cfg_id)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    seg = _seg_tensor(segs)
    a = sim.simulate(seg, rhat)
    blk = int(sim.dims.block_floats) * 4
    b = sim.simulate_chunked(seg, rhat, payload_budget_bytes=max(a["nblocks"] // 5, 1) * blk)
    assert b["chunks"] >= 3
    assert b["nblocks"] == a["nblocks"] and b["ntiles"] == a["ntiles"]
    assert torch.equal(a["tile_keys"], b["tile_keys"])
    assert torch.equal(a["tile_data"], b["tile_data"])
    # parity of the chunked result with the oracle on a few pixels
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    payload = o.effq(cfg, aug, keys)
    tiles = o.out_tiles(cfg, keys)
    act = np.unique(tiles % (cfg.npix_x * cfg.npix_y))
    pix = act[:: max(1, len(act) // 12)]
    ref = o.conv_fft(cfg, keys, payload, R, pix)
    c = sim.simulate_chunked(seg, rhat, pix_ids=torch.from_numpy(pix.astype(np.int32)).cuda(),
                             payload_budget_bytes=max(a["nblocks"] // 5, 1) * blk)
    _wave_checks(c["dense"].cpu().numpy().astype(np.float64), ref, sim.last_mac_mode())


# ------------------------------------------------------------------ N2: G4Step preprocessing
@pytest.mark.parametrize("model", [0, 1])
def test_steps_parity(model):
    """tred_steps vs the oracle: piece counts, parents and segment ends bit-exact (fp64
    round-to-nearest index path), electrons within 1e-6 (log / division rounding)."""
    torch = _torch()
    from paper_2602_12052_b200 import split_steps
    steps = gen.make_steps(21, n_tracks=30)
    par = dict(gen.STEP_PARAMS, recomb_model=model)
    ref = o.split_steps(par, steps)
    st = torch.from_numpy(np.ascontiguousarray(np.stack([steps[k] for k in gen.STEP_FIELDS]))).cuda()
    seg, parent, nseg = split_steps(st, par)
    assert int(nseg.item()) == len(ref["parent"])
    np.testing.assert_array_equal(parent.cpu().numpy(), ref["parent"])
    got = seg.cpu().numpy()
    for i, k in enumerate(gen.SEG_FIELDS):
        if k == "q":
            np.testing.assert_allclose(got[i], ref["segs"][k], rtol=1e-6)
        else:
            np.testing.assert_array_equal(got[i], ref["segs"][k], err_msg=k)
    # capacity semantics: too small a buffer still reports the count and stays in bounds
    seg2, parent2, nseg2 = split_steps(st, par, cap_seg=10)
    assert int(nseg2.item()) == len(ref["parent"]) and seg2.shape[1] == 10
    np.testing.assert_array_equal(seg2.cpu().numpy()[0], ref["segs"]["x0"][:10])
    # and the segments feed the hot path
    cfg = gen.make_config(2)
    sim = _sim(cfg)
    augf, augi, npairs = sim.drift(seg.contiguous())
    aug = o.drift(cfg, {k: got[i] for i, k in enumerate(gen.SEG_FIELDS)})
    np.testing.assert_array_equal(augi.cpu().numpy()[:6], np.concatenate([aug["lo"].T, aug["hi"].T]))


# ------------------------------------------------------------------ N3: trigger-reset readout
@pytest.mark.parametrize("with_noise", [False, True])
def test_readout_parity(with_noise):
    """tred_readout on the waveforms of the path (config 1) vs the oracle on the same fp32
    waveforms: hit counts, digitisation ticks and ADC words bit-exact (same fp32 running sum)."""
    torch = _torch()
    from paper_2602_12052_b200 import readout
    cfg, segs = _small(1)
    R = gen.make_response(cfg, 2001)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    pix = torch.arange(0, cfg.npix_x * cfg.npix_y, 3, dtype=torch.int32).cuda()
    wave = sim.simulate(_seg_tensor(segs), rhat, pix_ids=pix)["dense"]
    par = dict(threshold_e=3000.0, n_integ=16, n_reset=8, max_hits=12, adc_lsb_e=250.0 if with_noise else 0.0)
    noise = None
    if with_noise:      # discriminator 650 e, preamplifier 500 e, baseline 900 e
        rng = np.random.default_rng(99)
        noise = (rng.standard_normal((pix.numel(), par["max_hits"], 3)) * [650.0, 500.0, 900.0]).astype(np.float32)
    nh, tk, adc = readout(wave, par, None if noise is None else torch.from_numpy(noise).cuda())
    rn, rt, ra = o.readout(par, wave.cpu().numpy(), noise)
    assert rn.sum() > 20 and rn.max() >= 2                     # the track is seen, some pixels fire repeatedly
    np.testing.assert_array_equal(nh.cpu().numpy(), rn)
    np.testing.assert_array_equal(tk.cpu().numpy(), rt)
    np.testing.assert_array_equal(adc.cpu().numpy(), ra)
    # empty input and zero capacity
    z = torch.zeros((5, 64), dtype=torch.float32).cuda()
    assert int(readout(z, par)[0].sum()) == 0


def test_readout_full_plane():
    """All 230 x 230 channels x 5000 ticks of a config-3 plane (one vertex) in one call: channels the
    event never reaches record nothing; 150 of the busiest channels and 150 random active ones are
    bit-exact against the oracle (which walks a channel tick by tick in Python)."""
    torch = _torch()
    from paper_2602_12052_b200 import readout
    cfg, segs = gen.make_segments(3, n_vertices=1)
    R = gen.make_response(cfg, 2003)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    npix = cfg.npix_x * cfg.npix_y
    pix = torch.arange(npix, dtype=torch.int32, device="cuda")
    wave = sim.simulate(_seg_tensor(segs), rhat, pix_ids=pix)["dense"]
    assert tuple(wave.shape) == (npix, cfg.nticks)
    par = dict(threshold_e=4000.0, n_integ=16, n_reset=8, max_hits=24, adc_lsb_e=100.0)
    rng = np.random.default_rng(7)
    noise = (rng.standard_normal((npix, par["max_hits"], 3)) * [650.0, 500.0, 900.0]).astype(np.float32)
    nh, tk, adc = readout(wave, par, torch.from_numpy(noise).cuda())
    nh, tk, adc = nh.cpu().numpy(), tk.cpu().numpy(), adc.cpu().numpy()
    l1 = wave.abs().sum(1).cpu().numpy()
    silent = l1 == 0
    assert silent.sum() > 1000 and (nh[silent] == 0).all() and (tk[silent] == -1).all()
    assert nh.sum() > 5000 and nh.max() >= 4
    active = np.flatnonzero(~silent)
    sel = np.unique(np.concatenate([active[np.argsort(l1[active])[-150:]], rng.choice(active, 150, replace=False)]))
    rn, rt, ra = o.readout(par, wave[torch.from_numpy(sel).cuda()].cpu().numpy(), noise[sel])
    np.testing.assert_array_equal(nh[sel], rn)
    np.testing.assert_array_equal(tk[sel], rt)
    np.testing.assert_array_equal(adc[sel], ra)


# ------------------------------------------------------------------ full size (configs 3 and 4)
# Neighbourhoods checked against the oracle at full size (config 3; a quarter as many at config 4).
# The oracle needs about 10 s per neighbourhood on the 16+ host cores of a GPU box (every segment
# within the response's reach, all time slabs); TRED_FULL_NEIGHBOURHOODS changes the sample size.
NFULL = int(os.environ.get("TRED_FULL_NEIGHBOURHOODS", "16"))


def _check_neighbourhoods(cfg, aug, keys, R, groups, dense, mode, payload_rows=None):
    """Waveforms of every pixel group against the oracle run on the blocks within the response's
    reach of the group (only those contribute), and the effective charge of those blocks."""
    torch = _torch()
    g = o.grid_of(cfg)
    npy, S, H = cfg.npix_y, cfg.sub, cfg.resp_half
    bx, by, bt = o.key_to_bxyz(g, keys)
    Bx, By = cfg.block[0], cfg.block[1]
    row = 0
    for grp in groups:
        px, py = grp // npy, grp % npy
        m = ((Bx * bx + Bx - 1) // S >= px.min() - H) & ((Bx * bx) // S <= px.max() + H) & \
            ((By * by + By - 1) // S >= py.min() - H) & ((By * by) // S <= py.max() + H)
        kk = keys[m]
        sel = o.segments_touching(cfg, aug, kk)
        payload = o.effq(cfg, aug, kk, sel)
        ref = o.conv_fft(cfg, kk, payload, R, grp)
        _wave_checks(dense[row: row + len(grp)], ref, mode)
        row += len(grp)
        if payload_rows is not None:
            got_q = payload_rows[torch.from_numpy(np.flatnonzero(m)).cuda()].cpu().numpy().astype(np.float64)
            assert np.abs(got_q - payload).max() <= TOL_QEFF * np.abs(payload).max()


def _pick_groups(cfg, tiles, n, seed):
    npy = cfg.npix_y
    rng = np.random.default_rng(seed)
    act = np.unique(tiles % (cfg.npix_x * npy))
    inner = act[(act // npy > 8) & (act // npy < cfg.npix_x - 8) & (act % npy > 8) & (act % npy < npy - 8)]
    centres = rng.choice(inner, n, replace=False)
    return [np.array([c, c + npy], dtype=np.int64) for c in centres]


def test_full_size_config3_sampled_pixels():
    """BASELINE config 3 at full size, in the configuration bench.py times: all integer outputs
    (block keys, output tile keys) bit-exact in full; waveforms and effective charge on sampled
    pixel neighbourhoods, which the oracle can compute one at a time."""
    torch = _torch()
    cfg, segs = gen.make_segments(3)
    R = gen.make_response(cfg, 2003)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    tiles = o.out_tiles(cfg, keys)
    groups = _pick_groups(cfg, tiles, NFULL, 33)
    pix_all = np.concatenate(groups)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    out = sim.simulate(_seg_tensor(segs), rhat, torch.from_numpy(pix_all.astype(np.int32)).cuda(), keep=True)
    assert out["nblocks"] == len(keys)
    np.testing.assert_array_equal(out["keys"].cpu().numpy(), keys)
    np.testing.assert_array_equal(out["tile_keys"].cpu().numpy(), tiles)
    dense = out["dense"].cpu().numpy().astype(np.float64)
    _check_neighbourhoods(cfg, aug, keys, R, groups, dense, sim.last_mac_mode(), out["payload"])
    # the one-call path (tred_simulate) gives the same bits as the stepwise calls
    one = sim.simulate(_seg_tensor(segs), rhat, torch.from_numpy(pix_all.astype(np.int32)).cuda())
    assert torch.equal(one["tile_keys"], out["tile_keys"]) and torch.equal(one["dense"], out["dense"])


def test_full_size_config4_chunked():
    """BASELINE config 4 at full size (10 overlaid spills, ~10.5 M segments, 700 x 700 pixels), run as
    bench.py runs it: slab-range chunks under a 5 GiB payload budget and a 5 GiB convolution
    workspace.  The tile list is compared in full with the oracle's, the waveforms on sampled
    neighbourhoods (chunking must not change the result)."""
    torch = _torch()
    cfg, segs = gen.make_segments(4)
    R = gen.make_response(cfg, 2004)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    tiles = o.out_tiles(cfg, keys)
    groups = _pick_groups(cfg, tiles, max(1, NFULL // 4), 44)
    pix_all = np.concatenate(groups)
    sim = _sim(cfg, conv_work_bytes=5 << 30)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    torch.cuda.reset_peak_memory_stats()
    out = sim.simulate_chunked(_seg_tensor(segs), rhat, torch.from_numpy(pix_all.astype(np.int32)).cuda(),
                               payload_budget_bytes=5 << 30)
    torch.cuda.synchronize()
    assert out["chunks"] >= 9 and out["nblocks"] == len(keys)
    peak = torch.cuda.max_memory_allocated()
    assert peak <= 40e9, peak                                            # BASELINE: peak memory <= 40 GB
    np.testing.assert_array_equal(out["tile_keys"].cpu().numpy(), tiles)
    dense = out["dense"].cpu().numpy().astype(np.float64)
    _check_neighbourhoods(cfg, aug, keys, R, groups, dense, sim.last_mac_mode())


def test_dense_grid_equals_block_sparse():
    """BASELINE config 5's comparison point as a test: the convolution of the WHOLE plane on the dense
    grid (one 3-D FFT per sub-pixel phase, the paper's Eq. (14) as printed; torch.fft
    on the GPU as a library step of the check) equals the block-sparse result on every pixel of a
    reduced plane -- only blocks with activity matter."""
    torch = _torch()
    import bench
    cfg, segs = gen.make_segments(2)
    cfg = cfg.with_(npix_x=48, npix_y=40, nticks=1024)
    segs = {k: v[:1500].copy() for k, v in segs.items()}
    for a, n in (("x", cfg.npix_x), ("y", cfg.npix_y)):                 # fold the event into the small plane
        for e in ("0", "1"):
            segs[a + e] = np.mod(segs[a + e], n * cfg.pitch_mm * 0.98).astype(np.float32)
    for e in ("0", "1"):                                                  # ... and into the short time window
        segs["z" + e] = (10.0 + np.mod(segs["z" + e], 120.0)).astype(np.float32)
    keep = (np.abs(segs["x1"] - segs["x0"]) < 2.0) & (np.abs(segs["y1"] - segs["y0"]) < 2.0) & \
           (np.abs(segs["z1"] - segs["z0"]) < 2.0)                                               # not wrapped
    segs = {k: v[keep] for k, v in segs.items()}
    R = gen.make_random_response(cfg, 9)
    sim = _sim(cfg)
    R_d = torch.from_numpy(R).cuda()
    rhat = sim.prepare_response(R_d)
    pix = torch.arange(cfg.npix_x * cfg.npix_y, dtype=torch.int32, device="cuda")
    out = sim.simulate(_seg_tensor(segs), rhat, pix, keep=True)
    assert out["nblocks"] > 50
    rows, _, _ = bench.dense_grid_convolution(torch, cfg, out["keys"], out["payload"], R_d, pix)
    err = float((rows - out["dense"]).abs().max() / out["dense"].abs().max())
    assert err <= 2e-5, err


# ------------------------------------------------------------------ N4: truth attribution
def test_attribution_by_reconvolution():
    """waveform-level truth attribution re-convolves selected contributions.
    Per-group waveforms match the oracle run on that group alone, and add up to the whole."""
    torch = _torch()
    cfg, segs = _small(2)
    n = len(segs["q"])
    R = gen.make_response(cfg, 2002)
    group = (np.arange(n) * 3 // n).astype(np.int64)           # three "tracks": consecutive thirds
    group[::17] = -1                                            # some segments without a label
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    seg = _seg_tensor(segs)
    aug = o.drift(cfg, segs)
    tiles = o.out_tiles(cfg, o.blocks(cfg, aug))
    act = np.unique(tiles % (cfg.npix_x * cfg.npix_y))
    pix = act[:: max(1, len(act) // 10)][:10]
    pix_d = torch.from_numpy(pix.astype(np.int32)).cuda()
    per = sim.attribute(seg, rhat, torch.from_numpy(group).cuda(), pix_d).cpu().numpy().astype(np.float64)
    assert per.shape == (3, len(pix), cfg.nticks)
    for gid in range(3):
        sub = {k: v[group == gid] for k, v in segs.items()}
        ref = o.simulate(cfg, sub, R, pix=pix, fft=True)["wave"]
        scale = max(np.abs(ref).max(), 1e-30)
        assert np.abs(per[gid] - ref).max() <= TOL_WAVE * scale
    labelled = {k: v[group >= 0] for k, v in segs.items()}
    whole = sim.simulate(_seg_tensor(labelled), rhat, pix_ids=pix_d)["dense"].cpu().numpy().astype(np.float64)
    assert np.abs(per.sum(0) - whole).max() <= 5e-6 * np.abs(whole).max()


# ------------------------------------------------------------------ degenerate inputs
def test_empty_and_out_of_window_inputs():
    """No segments, and segments whose charge falls entirely outside the grid / time window
    (clip-and-drop, reading G13): no blocks, no tiles, zero waveforms, no error."""
    torch = _torch()
    cfg, segs = _small(1)
    R = gen.make_response(cfg, 2001)
    sim = _sim(cfg)
    rhat = sim.prepare_response(torch.from_numpy(R).cuda())
    pix = torch.arange(0, 16, dtype=torch.int32).cuda()
    empty = torch.empty((8, 0), dtype=torch.float32).cuda()
    out = sim.simulate(empty, rhat, pix_ids=pix)
    assert out["nblocks"] == 0 and out["ntiles"] == 0 and float(out["dense"].abs().max()) == 0.0
    far = {k: v[:50].copy() for k, v in segs.items()}
    far["x0"] += 1.0e4; far["x1"] += 1.0e4                    # 10 m off the pixel plane
    out = sim.simulate(_seg_tensor(far), rhat, pix_ids=pix)
    assert out["nblocks"] == 0 and out["ntiles"] == 0 and float(out["dense"].abs().max()) == 0.0
    assert len(o.blocks(cfg, o.drift(cfg, far))) == 0
    late = {k: v[:50].copy() for k, v in segs.items()}
    late["t0"] += 1.0e4                                        # arrives after the window
    out = sim.simulate(_seg_tensor(late), rhat, pix_ids=pix)
    assert out["nblocks"] == len(o.blocks(cfg, o.drift(cfg, late))) == 0
    # chunked driver on an empty event
    out = sim.simulate_chunked(empty, rhat, pix_ids=pix)
    assert out["ntiles"] == 0 and float(out["dense"].abs().max()) == 0.0


# ------------------------------------------------------------------ N4: truth record
@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_truth_record_parity(cfg_id):
    """tred_truth vs the oracle: (segment, key) lists bit-exact, charges within the
    effective-charge tolerance; capacity semantics."""
    torch = _torch()
    cfg, segs = _small(cfg_id)
    segs = {k: v[:60] for k, v in segs.items()}
    aug = o.drift(cfg, segs)
    rs, rk, rq = o.truth_record(cfg, aug)
    sim = _sim(cfg)
    augf, augi, _ = sim.drift(_seg_tensor(segs))
    gs, gk, gq, nrec = sim.truth(augf, augi)
    assert int(nrec.item()) == len(rs)
    np.testing.assert_array_equal(gs.cpu().numpy(), rs)
    np.testing.assert_array_equal(gk.cpu().numpy(), rk)
    got = gq.cpu().numpy().astype(np.float64)
    assert np.abs(got - rq).max() <= TOL_QEFF * np.abs(rq).max()
    tot_g = np.bincount(rs, weights=got, minlength=60)
    tot_r = np.bincount(rs, weights=rq, minlength=60)
    assert np.allclose(tot_g, tot_r, rtol=1e-5)
    gs2, gk2, gq2, nrec2 = sim.truth(augf, augi, cap_rec=7)
    assert int(nrec2.item()) == len(rs) and gs2.numel() == 7
    np.testing.assert_array_equal(gk2.cpu().numpy(), rk[:7])


def test_truth_long_segments_and_overflow():
    """A record holds up to 32 pixels / time tiles per axis: a 90 mm step far from the anode (about 60
    sigma long, 22 pixels) is booked in full and matches the oracle; a 200 mm step exceeds the record
    and is REPORTED (count -1), not truncated."""
    import paper_2602_12052_b200 as pkg
    cfg = gen.make_config(2)
    rows = [(100.0, 200.0, 400.0, 190.0, 203.0, 401.0, 5.4e5, 0.0),        # 90 mm along x
            (300.0, 100.0, 250.0, 300.5, 100.2, 290.0, 2.4e5, 0.0)]        # 40 mm along the drift: 250 ticks, 3 tiles
    segs = {k: np.array([r[i] for r in rows], np.float32) for i, k in enumerate(gen.SEG_FIELDS)}
    aug = o.drift(cfg, segs)
    rs, rk, rq = o.truth_record(cfg, aug)
    sim = _sim(cfg)
    augf, augi, _ = sim.drift(_seg_tensor(segs))
    gs, gk, gq, nrec = sim.truth(augf, augi)
    assert int(nrec.item()) == len(rs) and len(rs) > 60
    np.testing.assert_array_equal(gs.cpu().numpy(), rs)
    np.testing.assert_array_equal(gk.cpu().numpy(), rk)
    got = gq.cpu().numpy().astype(np.float64)
    assert np.abs(got - rq).max() <= TOL_QEFF * np.abs(rq).max()
    assert np.allclose(np.bincount(rs, weights=got), np.bincount(rs, weights=rq), rtol=1e-5)
    long = {k: np.array([(100.0, 200.0, 400.0, 300.0, 203.0, 401.0, 1.2e6, 0.0)[i]], np.float32)
            for i, k in enumerate(gen.SEG_FIELDS)}
    augf, augi, _ = sim.drift(_seg_tensor(long))
    with pytest.raises(pkg.TredError):
        sim.truth(augf, augi)
