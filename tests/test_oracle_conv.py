"""Pins of the oracle's interlaced convolution (O5, Eq. 12/14).  CPU only."""
import numpy as np
from scipy import signal

import gen
import oracle as o


def _cfg(**kw):
    base = dict(npix_x=14, npix_y=13, nticks=96, gl_n=2, block=(8, 8, 32), resp_nticks=24)
    base.update(kw)
    return gen.make_config(1, **base)


def _payload_from_dense(cfg, dense):
    """Cut a dense fine-grid array into the block list of its non-zero blocks."""
    g = o.grid_of(cfg)
    pad = np.zeros(tuple(g.NB[a] * g.B[a] for a in range(3)))
    pad[:g.NG[0], :g.NG[1], :g.NG[2]] = dense
    keys, tiles = [], []
    for bt in range(g.NB[2]):
        for bx in range(g.NB[0]):
            for by in range(g.NB[1]):
                t = pad[bx*g.B[0]:(bx+1)*g.B[0], by*g.B[1]:(by+1)*g.B[1], bt*g.B[2]:(bt+1)*g.B[2]]
                if np.any(t != 0):
                    keys.append((bt * g.NB[0] + bx) * g.NB[1] + by)
                    tiles.append(t.copy())
    return np.array(keys, np.int64), np.array(tiles)


def test_impulse_returns_the_response_at_its_phase_and_offsets():
    """Eq. (12) with Qeff = delta at fine column (i,j), tick t0: the waveform on pixel
    (Px+kx, Py+ky) is R[jx, jy, kx, ky, t - t0] (readings G3, G12: source->output
    displacement, causal).  An unstructured random response pins every index."""
    cfg = _cfg()
    R = gen.make_random_response(cfg, 3)
    S, H = cfg.sub, cfg.resp_half
    g = o.grid_of(cfg)
    dense = np.zeros(g.NG)
    i, j, t0 = 6 * S + 3, 7 * S + 8, 17                    # pixel (6,7), phase (3,8)
    dense[i, j, t0] = 2.5
    keys, payload = _payload_from_dense(cfg, dense)
    pix = np.arange(cfg.npix_x * cfg.npix_y)
    for conv in (o.conv_direct, o.conv_fft):
        w = conv(cfg, keys, payload, R, pix).reshape(cfg.npix_x, cfg.npix_y, -1)
        for kx in range(-H, H + 1):
            for ky in range(-H, H + 1):
                px, py = 6 + kx, 7 + ky
                ref = np.zeros(cfg.nticks)
                ref[t0:t0 + cfg.resp_nticks] = 2.5 * R[3, 8, kx + H, ky + H].astype(np.float64)
                np.testing.assert_allclose(w[px, py], ref, atol=1e-12)
        far = np.ones((cfg.npix_x, cfg.npix_y), bool)
        far[1:12, 2:13] = False
        assert np.abs(w[far]).max() < 1e-12


def test_against_scipy_convolve_per_phase():
    """Independent library route: for every phase (jx,jy) the pixel-plane x time
    array Q^j[Px,Py,t] is convolved with R[jx,jy,:,:,:] by scipy.signal.convolve
    ('full', direct method) -- PAPER.md Eq. (12) read literally as a 3-D convolution
    per sub-pixel offset j followed by the sum over j."""
    cfg = _cfg(npix_x=6, npix_y=7, nticks=40, resp_nticks=9, resp_half=2, block=(4, 4, 8))
    S, H, Tr = cfg.sub, cfg.resp_half, cfg.resp_nticks
    R = gen.make_random_response(cfg, 4)
    g = o.grid_of(cfg)
    rng = np.random.default_rng(5)
    dense = np.zeros(g.NG)
    idx = rng.integers(0, [g.NG[0], g.NG[1], g.NG[2]], size=(60, 3))
    dense[idx[:, 0], idx[:, 1], idx[:, 2]] = rng.standard_normal(60)
    keys, payload = _payload_from_dense(cfg, dense)
    pix = np.arange(cfg.npix_x * cfg.npix_y)
    got = o.conv_direct(cfg, keys, payload, R, pix).reshape(cfg.npix_x, cfg.npix_y, -1)
    Qj = dense.reshape(cfg.npix_x, S, cfg.npix_y, S, -1)
    ref = np.zeros((cfg.npix_x + 2 * H, cfg.npix_y + 2 * H, cfg.nticks + Tr - 1))
    for jx in range(S):
        for jy in range(S):
            ref += signal.convolve(Qj[:, jx, :, jy, :], R[jx, jy].astype(np.float64),
                                   mode="full", method="direct")
    ref = ref[H:H + cfg.npix_x, H:H + cfg.npix_y, :cfg.nticks]
    np.testing.assert_allclose(got, ref, atol=1e-11)
    got_fft = o.conv_fft(cfg, keys, payload, R, pix).reshape(got.shape)
    np.testing.assert_allclose(got_fft, ref, atol=1e-11)


def test_fft_matches_direct_on_a_track_and_is_linear():
    cfg, segs = gen.make_segments(1)
    segs = {k: v[:30] for k, v in segs.items()}
    R = gen.make_response(cfg, 2001)
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    payload = o.effq(cfg, aug, keys)
    rng = np.random.default_rng(1)
    pix = np.sort(rng.choice(cfg.npix_x * cfg.npix_y, 24, replace=False))
    a = o.conv_direct(cfg, keys, payload, R, pix)
    b = o.conv_fft(cfg, keys, payload, R, pix)
    assert np.abs(a).max() > 0
    assert np.abs(a - b).max() < 1e-10 * np.abs(a).max()
    c = o.conv_direct(cfg, keys, 3.0 * payload, R, pix)
    np.testing.assert_allclose(c, 3.0 * a, rtol=1e-12, atol=1e-9)


def test_shift_equivariance_whole_pixel_and_tick():
    """Shifting Qeff by one pixel (S fine points) / one tick shifts the output."""
    cfg = _cfg()
    R = gen.make_random_response(cfg, 6)
    g = o.grid_of(cfg)
    S = cfg.sub
    rng = np.random.default_rng(2)
    dense = np.zeros(g.NG)
    dense[50:70, 40:65, 20:40] = rng.standard_normal((20, 25, 20))
    pix = np.arange(cfg.npix_x * cfg.npix_y)
    k0, p0 = _payload_from_dense(cfg, dense)
    w0 = o.conv_fft(cfg, k0, p0, R, pix).reshape(cfg.npix_x, cfg.npix_y, -1)
    sh = np.zeros_like(dense)
    sh[S:, :-S, 2:] = dense[:-S, S:, :-2]                 # +1 pixel x, -1 pixel y, +2 ticks
    k1, p1 = _payload_from_dense(cfg, sh)
    w1 = o.conv_fft(cfg, k1, p1, R, pix).reshape(cfg.npix_x, cfg.npix_y, -1)
    # compare where neither version was clipped by the plane / window
    np.testing.assert_allclose(w1[1:, :-1, 2:], w0[:-1, 1:, :-2], atol=1e-10)


def test_per_pixel_integral_equals_collected_charge():
    """Reading G18: the synthetic response integrates to 1 on the collecting pixel and
    0 elsewhere, so sum_t I_p(t) = sum of Qeff inside pixel p (untruncated window)."""
    cfg = _cfg(nticks=160, resp_nticks=40)
    R = gen.make_response(cfg, 2001)
    g = o.grid_of(cfg)
    S = cfg.sub
    rng = np.random.default_rng(3)
    dense = np.zeros(g.NG)
    dense[40:90, 30:100, 10:60] = rng.uniform(0, 1, (50, 70, 50))
    keys, payload = _payload_from_dense(cfg, dense)
    pix = np.arange(cfg.npix_x * cfg.npix_y)
    w = o.conv_fft(cfg, keys, payload, R, pix).reshape(cfg.npix_x, cfg.npix_y, -1)
    qpix = dense.reshape(cfg.npix_x, S, cfg.npix_y, S, -1).sum((1, 3, 4))
    # R is cast to fp32 (rounding ~6e-8 per sample, 121 x 100 phases feed one pixel)
    np.testing.assert_allclose(w.sum(2), qpix, atol=2e-5 * qpix.max())


def test_response_recipe_properties():
    """DESIGN.md input recipe: unit integral on the centre pixel, zero elsewhere,
    reflection symmetry R_{-i}^{-j} = R_i^j."""
    cfg = gen.make_config(1)
    R = gen.make_response(cfg, 2001).astype(np.float64)
    H = cfg.resp_half
    s = R.sum(-1)
    assert np.abs(s[:, :, H, H] - 1).max() < 1e-5
    s[:, :, H, H] = 0
    assert np.abs(s).max() < 1e-5
    np.testing.assert_array_equal(R, R[::-1, ::-1, ::-1, ::-1, :])
