"""TRED hot-path ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain, slow, fp64 CPU restatement of the data-parallel hot path of
arxiv 2602.12052, written from the paper and from the readings
listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's
`cpu_baseline` / `--impl reference` legs may import this package.  It shares
no code with paper_2602_12052_b200/ (the CUDA path) and never imports it.

Steps (names follow SURVEY.md Sec. 8(c)):
  O1 drift()        PAPER.md:L41,L57 (attachment, drift, diffusion width)
  O2 charge density PAPER.md:L128-148, Eq. (10)         -> tred_oracle.c
  O3 effq()         PAPER.md:L85-126,L197, Eq. (9)      -> tred_oracle.c
  O4 blocks()       PAPER.md:L57,L236-240 (block-sparse binned tensor)
  O5 conv_direct()  PAPER.md:L150-173, Eq. (12), direct sum -> tred_oracle.c
     conv_fft()     PAPER.md:L223-228, Eq. (14) with numpy's FFT (library step)
  O6 out_tiles()    PAPER.md:L240,L250 (footprint of the output)

Parity pins: tests/test_oracle_*.py.  Unpinned: the magnitudes of Fig. 7
(their response and data are not available) -- only the
ordering err(n=1) > err(n=2) is checked; the paper's runtimes (context only).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(_build.build())
        _LIB.tred_o_q.restype = ctypes.c_double
    return _LIB


class _CGrid(ctypes.Structure):
    _fields_ = [("NG", ctypes.c_int64 * 3), ("B", ctypes.c_int64 * 3),
                ("NB", ctypes.c_int64 * 3), ("org", ctypes.c_double * 3),
                ("h", ctypes.c_double * 3)]


@dataclass
class Grid:
    NG: tuple      # fine-grid points (x, y, t)
    B: tuple       # block shape
    NB: tuple      # blocks per axis
    org: tuple     # origin (x, y, t)
    h: tuple       # spacing (hx, hy, dt)

    def c(self) -> _CGrid:
        g = _CGrid()
        for i in range(3):
            g.NG[i], g.B[i], g.NB[i] = self.NG[i], self.B[i], self.NB[i]
            g.org[i], g.h[i] = self.org[i], self.h[i]
        return g


def grid_of(cfg) -> Grid:
    """Fine grid G: pixel pitch / S by time tick."""
    NG = (cfg.sub * cfg.npix_x, cfg.sub * cfg.npix_y, cfg.nticks)
    B = tuple(int(b) for b in cfg.block)
    NB = tuple(-(-NG[i] // B[i]) for i in range(3))
    hxy = cfg.pitch_mm / cfg.sub
    return Grid(NG, B, NB, (cfg.origin_x_mm, cfg.origin_y_mm, cfg.t_origin_us),
                (hxy, hxy, cfg.tick_us))


# ---------------------------------------------------------------------------
# quadrature constants
# ---------------------------------------------------------------------------
def gl_rule(n: int):
    """Nodes/weights of the n-point Gauss-Legendre rule on [-1,1]."""
    xi, w = np.polynomial.legendre.leggauss(n)
    return xi.astype(np.float64), w.astype(np.float64)


def trilinear_u(xi: np.ndarray) -> np.ndarray:
    """1-D factors of u_{lmn,rst} (Eq. (7)); u[l, r+1], r=-1,0,+1.
    A node at offset xi/2 (in cuboid widths) from the cuboid centre interpolates
    linearly between its own grid point and the neighbour on its side."""
    u = np.zeros((len(xi), 3))
    u[:, 0] = np.maximum(-xi, 0.0) / 2.0
    u[:, 1] = 1.0 - np.abs(xi) / 2.0
    u[:, 2] = np.maximum(xi, 0.0) / 2.0
    return u


# ---------------------------------------------------------------------------
# O1 drift
# ---------------------------------------------------------------------------
def drift(cfg, segs) -> dict:
    """Arrival times, attenuated charge, diffusion widths, point/line flag and
    the integer cuboid bounding box of every segment.

    The *index path* (everything that decides an integer) is fp64 with this
    exact operation order, no contraction (reading G14)."""
    f = lambda k: np.asarray(segs[k], dtype=np.float64)
    x0, y0, z0, x1, y1, z1, q, t0 = (f(k) for k in ("x0", "y0", "z0", "x1", "y1", "z1", "q", "t0"))
    g = grid_of(cfg)
    v = np.float64(cfg.v_mm_us)
    ta0 = t0 + z0 / v
    ta1 = t0 + z1 / v
    tm = (z0 + z1) / (np.float64(2.0) * v)
    tmc = np.maximum(tm, 0.0)
    sxy = np.maximum(np.sqrt((np.float64(2.0) * np.float64(cfg.DT_mm2_us)) * tmc),
                     np.float64(cfg.sigma_min_xy_mm))
    st = np.maximum(np.sqrt((np.float64(2.0) * np.float64(cfg.DL_mm2_us)) * tmc) / v,
                    np.float64(cfg.sigma_min_t_us))
    Qp = q * np.exp(-tm / np.float64(cfg.lifetime_us))
    pt = np.float64(cfg.point_thresh)
    flag = ((np.abs(x1 - x0) < pt * sxy) & (np.abs(y1 - y0) < pt * sxy)
            & (np.abs(ta1 - ta0) < pt * st))
    ns = np.float64(cfg.nsigma)
    mxy, mt = ns * sxy, ns * st

    def box(a0, a1, m, org, h):
        lo = np.floor(((np.minimum(a0, a1) - m) - np.float64(org)) / np.float64(h))
        hi = np.floor(((np.maximum(a0, a1) + m) - np.float64(org)) / np.float64(h))
        return lo.astype(np.int64), hi.astype(np.int64)

    lox, hix = box(x0, x1, mxy, g.org[0], g.h[0])
    loy, hiy = box(y0, y1, mxy, g.org[1], g.h[1])
    lot, hit = box(ta0, ta1, mt, g.org[2], g.h[2])
    return dict(p0=np.stack([x0, y0, ta0], 1), p1=np.stack([x1, y1, ta1], 1),
                sig=np.stack([sxy, sxy, st], 1), Qp=Qp, tm=tm,
                flag=flag.astype(np.int32),
                lo=np.stack([lox, loy, lot], 1), hi=np.stack([hix, hiy, hit], 1))


# ---------------------------------------------------------------------------
# O4 blocks
# ---------------------------------------------------------------------------
def block_ranges(cfg, aug):
    """Per segment: inclusive block range [blo, bhi] per axis of the grid-point
    footprint [lo-e, hi+e] (e = 1 if n > 1 else 0) clipped to the grid, and a
    mask of segments whose clipped footprint is non-empty."""
    g = grid_of(cfg)
    e = 1 if cfg.gl_n > 1 else 0
    NG = np.array(g.NG, dtype=np.int64)
    B = np.array(g.B, dtype=np.int64)
    flo = np.maximum(aug["lo"] - e, 0)
    fhi = np.minimum(aug["hi"] + e, NG[None, :] - 1)
    ok = np.all(flo <= fhi, axis=1)
    return flo // B, fhi // B, ok


def block_key(g: Grid, bx, by, bt):
    """key = (bt*NBx + bx)*NBy + by : time slab major (reading G16)."""
    return (np.asarray(bt, np.int64) * g.NB[0] + bx) * g.NB[1] + by


def block_pairs(cfg, aug):
    """All (segment, block key) pairs, segment-major."""
    g = grid_of(cfg)
    blo, bhi, ok = block_ranges(cfg, aug)
    cnt = np.where(ok, np.prod(bhi - blo + 1, axis=1), 0)
    seg = np.repeat(np.arange(len(cnt), dtype=np.int64), cnt)
    start = np.cumsum(cnt) - cnt
    r = np.arange(int(cnt.sum()), dtype=np.int64) - np.repeat(start, cnt)
    nx = (bhi - blo + 1)[seg, 0]; ny = (bhi - blo + 1)[seg, 1]
    bt = blo[seg, 2] + r // (nx * ny)
    rem = r % (nx * ny)
    bx = blo[seg, 0] + rem // ny
    by = blo[seg, 1] + rem % ny
    return seg, block_key(g, bx, by, bt), cnt


def blocks(cfg, aug) -> np.ndarray:
    """Sorted unique keys of the occupied blocks (occupancy by footprint, G15)."""
    _, keys, _ = block_pairs(cfg, aug)
    return np.unique(keys)


def key_to_bxyz(g: Grid, keys):
    keys = np.asarray(keys, np.int64)
    by = keys % g.NB[1]
    bx = (keys // g.NB[1]) % g.NB[0]
    bt = keys // (g.NB[1] * g.NB[0])
    return bx, by, bt


def _blockslot(g: Grid, keys) -> np.ndarray:
    m = np.full(g.NB[0] * g.NB[1] * g.NB[2], -1, dtype=np.int64)
    m[np.asarray(keys, np.int64)] = np.arange(len(keys), dtype=np.int64)
    return m


# ---------------------------------------------------------------------------
# O2 / O3 effective charge
# ---------------------------------------------------------------------------
def charge_density(aug, s: int, pos) -> float:
    """Eq. (10) (corrected exponent) / point branch for segment s at pos=(x,y,t)."""
    d = lambda a: np.ascontiguousarray(a, np.float64).ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    return _lib().tred_o_q(d(aug["p0"][s]), d(aug["p1"][s]), d(aug["sig"][s]),
                           ctypes.c_double(float(aug["Qp"][s])), ctypes.c_int(int(aug["flag"][s])),
                           d(np.asarray(pos, np.float64)))


def effq(cfg, aug, keys, seg_select=None) -> np.ndarray:
    """Effective charge Eq. (9) restricted to the blocks `keys` (sorted unique).
    Returns payload [nblk][Bx][By][Bt] fp64.  `seg_select`: optional index array
    of the segments to process (e.g. those touching `keys`)."""
    g = grid_of(cfg)
    keys = np.asarray(keys, np.int64)
    xi, w = gl_rule(cfg.gl_n)
    u = trilinear_u(xi)
    payload = np.zeros((len(keys),) + g.B, dtype=np.float64)
    slot = _blockslot(g, keys)
    sel = np.arange(len(aug["Qp"])) if seg_select is None else np.asarray(seg_select)
    c = lambda a, t: np.ascontiguousarray(a[sel], dtype=t)
    p0, p1, sig = c(aug["p0"], np.float64), c(aug["p1"], np.float64), c(aug["sig"], np.float64)
    Qp, fl = c(aug["Qp"], np.float64), c(aug["flag"], np.int32)
    lo, hi = c(aug["lo"], np.int64), c(aug["hi"], np.int64)
    cg = g.c()
    P = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    _lib().tred_o_effq(ctypes.byref(cg), ctypes.c_int64(len(sel)), P(p0), P(p1), P(sig), P(Qp), P(fl),
                       P(lo), P(hi), ctypes.c_int(cfg.gl_n), P(xi), P(w), P(np.ascontiguousarray(u)),
                       P(slot), P(payload))
    return payload


def segments_touching(cfg, aug, keys) -> np.ndarray:
    """Indices of the segments whose footprint meets any of the blocks `keys`."""
    seg, pk, _ = block_pairs(cfg, aug)
    return np.unique(seg[np.isin(pk, np.asarray(keys, np.int64))])


def payload_to_dense(cfg, keys, payload) -> np.ndarray:
    g = grid_of(cfg)
    full = np.zeros(tuple(g.NB[i] * g.B[i] for i in range(3)), dtype=payload.dtype)
    bx, by, bt = key_to_bxyz(g, keys)
    for s in range(len(keys)):
        full[bx[s]*g.B[0]:(bx[s]+1)*g.B[0], by[s]*g.B[1]:(by[s]+1)*g.B[1],
             bt[s]*g.B[2]:(bt[s]+1)*g.B[2]] = payload[s]
    return full[:g.NG[0], :g.NG[1], :g.NG[2]]


# ---------------------------------------------------------------------------
# O5 convolution
# ---------------------------------------------------------------------------
def conv_direct(cfg, keys, payload, R, pix) -> np.ndarray:
    """Eq. (12) by direct summation for the pixels `pix` (flat ids px*Npy+py).
    Returns [len(pix)][Nt] fp64.  R: float32 [S][S][2H+1][2H+1][Tr]."""
    g = grid_of(cfg)
    keys = np.asarray(keys, np.int64)
    pix = np.ascontiguousarray(pix, np.int64)
    R = np.ascontiguousarray(R, np.float32)
    payload = np.ascontiguousarray(payload, np.float64)
    out = np.zeros((len(pix), g.NG[2]), dtype=np.float64)
    slot = _blockslot(g, keys)
    cg = g.c()
    P = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    I = ctypes.c_int64
    _lib().tred_o_conv_direct(ctypes.byref(cg), I(cfg.sub), I(cfg.resp_half), I(cfg.resp_nticks),
                              I(cfg.npix_x), I(cfg.npix_y), P(slot), P(payload), P(R),
                              I(len(pix)), P(pix), P(out))
    return out


def conv_fft(cfg, keys, payload, R, pix) -> np.ndarray:
    """Eq. (14): the same sum as conv_direct with the time convolution done by
    numpy's real FFT over the whole (zero-padded) readout window; the FFT is a
    library step.  Checked against conv_direct in tests/test_oracle_conv.py."""
    g = grid_of(cfg)
    S, H, Tr, Nt = cfg.sub, cfg.resp_half, cfg.resp_nticks, g.NG[2]
    bx, by, bt = key_to_bxyz(g, keys)
    cols = {}
    for s in range(len(keys)):
        cols.setdefault((int(bx[s]), int(by[s])), []).append((int(bt[s]), s))
    n = 1
    while n < Nt + Tr - 1:
        n *= 2
    qcache = {}

    def qhat(i, j):
        if (i, j) not in qcache:
            b = (i // g.B[0], j // g.B[1])
            if b not in cols:
                qcache[(i, j)] = None
            else:
                series = np.zeros(g.NB[2] * g.B[2])
                for (tb, s) in cols[b]:
                    series[tb*g.B[2]:(tb+1)*g.B[2]] = payload[s, i - b[0]*g.B[0], j - b[1]*g.B[1], :]
                qcache[(i, j)] = np.fft.rfft(series[:Nt], n)
        return qcache[(i, j)]

    out = np.zeros((len(pix), Nt))
    for ip, p in enumerate(np.asarray(pix, np.int64)):
        px, py = int(p) // cfg.npix_y, int(p) % cfg.npix_y
        acc = np.zeros(n // 2 + 1, dtype=np.complex128)
        for kx in range(-H, H + 1):
            for ky in range(-H, H + 1):
                cpx, cpy = px - kx, py - ky
                if not (0 <= cpx < cfg.npix_x and 0 <= cpy < cfg.npix_y):
                    continue
                for jx in range(S):
                    for jy in range(S):
                        qh = qhat(cpx * S + jx, cpy * S + jy)
                        if qh is None:
                            continue
                        acc += qh * np.fft.rfft(R[jx, jy, kx + H, ky + H].astype(np.float64), n)
        out[ip] = np.fft.irfft(acc, n)[:Nt]
    return out


# ---------------------------------------------------------------------------
# O6 output tiles
# ---------------------------------------------------------------------------
def out_tiles(cfg, keys) -> np.ndarray:
    """Sorted unique keys (tb*Npx + px)*Npy + py of the output tiles
    (pixel, Tt=Bt ticks) met by the output footprint of any occupied block:
    pixels [floor(Bx bx / S) - H, floor((Bx bx + Bx - 1)/S) + H],
    ticks [Bt bt, Bt bt + Bt + Tr - 2], clipped to the readout."""
    g = grid_of(cfg)
    S, H, Tr = cfg.sub, cfg.resp_half, cfg.resp_nticks
    bx, by, bt = key_to_bxyz(g, keys)
    ntb = -(-g.NG[2] // g.B[2])
    mask = np.zeros((ntb, cfg.npix_x, cfg.npix_y), dtype=bool)
    for s in range(len(keys)):
        x0 = max((g.B[0] * bx[s]) // S - H, 0)
        x1 = min((g.B[0] * bx[s] + g.B[0] - 1) // S + H, cfg.npix_x - 1)
        y0 = max((g.B[1] * by[s]) // S - H, 0)
        y1 = min((g.B[1] * by[s] + g.B[1] - 1) // S + H, cfg.npix_y - 1)
        t0 = g.B[2] * bt[s]
        t1 = min(g.B[2] * bt[s] + g.B[2] + Tr - 2, g.NG[2] - 1)
        mask[t0 // g.B[2]: t1 // g.B[2] + 1, x0:x1 + 1, y0:y1 + 1] = True
    return np.flatnonzero(mask.ravel()).astype(np.int64)


# ---------------------------------------------------------------------------
# whole path
# ---------------------------------------------------------------------------
def simulate(cfg, segs, R, pix=None, keys_select=None, fft=False) -> dict:
    """Segments in, per-pixel current waveforms out (Fig. 1).
    `pix`: flat pixel ids to evaluate (default: all).  `keys_select`: evaluate
    the charge only in these blocks (waveforms then see only their charge)."""
    aug = drift(cfg, segs)
    keys = blocks(cfg, aug)
    kk = keys if keys_select is None else np.asarray(keys_select, np.int64)
    sel = None if keys_select is None else segments_touching(cfg, aug, kk)
    payload = effq(cfg, aug, kk, sel)
    if pix is None:
        pix = np.arange(cfg.npix_x * cfg.npix_y, dtype=np.int64)
    wave = (conv_fft if fft else conv_direct)(cfg, kk, payload, R, pix)
    return dict(aug=aug, keys=keys, payload_keys=kk, payload=payload, pix=np.asarray(pix),
                wave=wave, tiles=out_tiles(cfg, keys))


# ---------------------------------------------------------------------------
# N2: G4Step preprocessing -- PAPER.md:L57 (splitting) and
# PAPER.md:L41,L57 (electrons surviving recombination).  Readings G21, G22 of DESIGN.md:
#   G21  a step longer than max_len is cut into n = ceil(len / max_len) pieces of EQUAL length
#        (all <= max_len); every piece keeps dE/dx, its dE is dE * (1 / n); shorter steps are
#        kept unchanged.
#   G22  "parameterized models of recombination" without a formula: the caller
#        picks Birks' law  R = A / (1 + k/(rho E) dE/dx)  or the modified box model
#        R = ln(alpha + b dE/dx) / (b dE/dx), b = beta/(rho E), clipped to [0, 1];
#        N_e = dE / W_ion * R.
# Units: mm, MeV (dE), MeV/cm (dE/dx), kV/cm, g/cm^3, eV (W_ion).
# ---------------------------------------------------------------------------
STEP_FIELDS = ("x0", "y0", "z0", "x1", "y1", "z1", "dE", "t0")


def recombination(par, dedx):
    """Surviving fraction R for dE/dx in MeV/cm (float64 array)."""
    dedx = np.asarray(dedx, dtype=np.float64)
    rhoE = par["density_g_cm3"] * par["efield_kv_cm"]
    if par["recomb_model"] == 0:                      # Birks
        return par["birks_A"] / (1.0 + par["birks_k"] / rhoE * dedx)
    x = par["box_beta"] / rhoE * dedx                 # modified box
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.log(par["box_alpha"] + x) / x
    r = np.where(x > 0.0, r, 0.0)
    return np.clip(r, 0.0, 1.0)


def split_steps(par, steps) -> dict:
    """G4Steps -> step-segments of at most max_len_mm with their ionisation electrons.
    Returns the segment SoA of drift() (x0..z1, q, t0 as float32), `parent` (int32 step
    index of every segment) and `count` (int32 pieces per step)."""
    p0 = np.stack([steps[k].astype(np.float64) for k in ("x0", "y0", "z0")], 1)
    p1 = np.stack([steps[k].astype(np.float64) for k in ("x1", "y1", "z1")], 1)
    d = p1 - p0
    length = np.sqrt((d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2])
    count = np.maximum(np.ceil(length / par["max_len_mm"]), 1.0).astype(np.int32)
    dE = steps["dE"].astype(np.float64)
    dedx = np.where(length > 0.0, dE / np.where(length > 0.0, length, 1.0) * 10.0, 0.0)   # MeV/cm
    ne = dE * 1.0e6 / par["w_ion_ev"] * recombination(par, dedx)                        # electrons per step
    parent = np.repeat(np.arange(len(count), dtype=np.int32), count)
    first = np.cumsum(count) - count
    k = (np.arange(len(parent)) - first[parent]).astype(np.float64)
    n = count[parent].astype(np.float64)
    fa, fb = k / n, (k + 1.0) / n
    out = {}
    for a, name in enumerate(("x", "y", "z")):
        out[name + "0"] = (p0[parent, a] + d[parent, a] * fa).astype(np.float32)
        out[name + "1"] = (p0[parent, a] + d[parent, a] * fb).astype(np.float32)
    out["q"] = (ne[parent] / n).astype(np.float32)
    out["t0"] = steps["t0"][parent].astype(np.float32)
    return dict(segs=out, parent=parent, count=count)


# ---------------------------------------------------------------------------
# N3: trigger-reset pixel readout -- PAPER.md:L185, L189 (Fig. 4), noise
# terms PAPER.md:L262.  Reading G23 of DESIGN.md (the paper gives the scheme in words only):
# per channel, tick by tick, in the kernel's precision (fp32 running sum, because the
# crossing tick is an integer decided by a floating-point comparison):
#   WAIT   q += I[t]; when q >= threshold + d_thr[h] the discriminator fires at tick tc = t;
#   INTEG  q += I[t] for the next n_integ ticks; at ts = tc + n_integ the record
#          (ts, q + d_adc[h]) is written (hits whose ts falls outside the window are lost);
#   RESET  q = d_base[h]; the n_reset ticks after ts are dead (their charge is dropped);
# d_thr, d_adc, d_base are the discriminator, preamplifier and baseline noise draws of hit h
# (inputs; zeros if absent).  adc_lsb_e > 0 rounds the record to that many electrons.
# ---------------------------------------------------------------------------
def readout(par, wave, noise=None):
    """wave [npix][nticks] float32 (electrons per tick) -> (nhit [npix] int32,
    tick [npix][max_hits] int32 (-1 where unused), adc [npix][max_hits] float32)."""
    wave = np.asarray(wave, dtype=np.float32)
    npix, nticks = wave.shape
    mh = int(par["max_hits"])
    nhit = np.zeros(npix, np.int32)
    tick = np.full((npix, mh), -1, np.int32)
    adc = np.zeros((npix, mh), np.float32)
    thr0 = np.float32(par["threshold_e"])
    lsb = np.float32(par.get("adc_lsb_e", 0.0))
    for p in range(npix):
        q = np.float32(0.0)
        h = 0
        state, left = 0, 0                                # 0 WAIT, 1 INTEG, 2 DEAD
        nz = (lambda k: np.float32(noise[p, h, k])) if noise is not None else (lambda k: np.float32(0.0))
        thr = np.float32(thr0 + nz(0)) if h < mh else thr0
        row = wave[p]
        for t in range(nticks):
            if h >= mh:
                break
            if state == 2:
                left -= 1
                if left == 0:
                    state = 0
                continue
            q = np.float32(q + row[t])
            fire = False
            if state == 0:
                if q >= thr:
                    if par["n_integ"] == 0:
                        fire = True
                    else:
                        state, left = 1, int(par["n_integ"])
            else:
                left -= 1
                fire = left == 0
            if fire:
                v = np.float32(q + nz(1))
                if lsb > 0:
                    v = np.float32(np.floor(np.float32(v / lsb) + np.float32(0.5)) * lsb)
                tick[p, h], adc[p, h] = t, v
                q = nz(2)
                h += 1
                nhit[p] = h
                if h < mh:
                    thr = np.float32(thr0 + nz(0))
                state, left = (2, int(par["n_reset"])) if par["n_reset"] > 0 else (0, 0)
    return nhit, tick, adc


# ---------------------------------------------------------------------------
# N4: truth record -- PAPER.md:L352-354 ("segment-id -> charge per
# (channel, short time slice)").  Reading G24 of DESIGN.md: the record of segment s is its
# effective charge (Eq. (9)) summed over the grid points of every pixel and every time tile
# of Bt ticks it reaches, one entry per (pixel, tile) of the clipped integer footprint
# [lo - e, hi + e] (entries at the rim of the footprint may hold tiny values), ordered by
# segment, then by the tile key (tb * npix_x + px) * npix_y + py.
# ---------------------------------------------------------------------------
def truth_record(cfg, aug, segs_sel=None):
    """Returns (seg [n] int32, key [n] int64, charge [n] float64)."""
    g = grid_of(cfg)
    e = 1 if cfg.gl_n > 1 else 0
    S, Bt = cfg.sub, cfg.block[2]
    nseg = len(aug["Qp"]) if "Qp" in aug else aug["lo"].shape[0]
    sel = range(nseg) if segs_sel is None else segs_sel
    rs, rk, rq = [], [], []
    all_keys = None
    for s in sel:
        lo = np.maximum(aug["lo"][s] - e, 0)
        hi = np.minimum(aug["hi"][s] + e, np.array(g.NG) - 1)
        if np.any(lo > hi):
            continue
        # this segment alone, on the blocks it touches
        sub = {k: (v[s:s + 1] if hasattr(v, "shape") and v.shape[:1] == (nseg,) else v) for k, v in aug.items()}
        keys_s = blocks(cfg, sub)
        pay = effq(cfg, sub, keys_s)
        bx, by, bt = key_to_bxyz(g, keys_s)
        Bx, By = cfg.block[0], cfg.block[1]
        acc = {}
        for b in range(len(keys_s)):
            i = Bx * bx[b] + np.arange(Bx)
            j = By * by[b] + np.arange(By)
            k = Bt * bt[b] + np.arange(Bt)
            for px in np.unique(i // S):
                mi = (i // S == px) & (i >= lo[0]) & (i <= hi[0])
                for py in np.unique(j // S):
                    mj = (j // S == py) & (j >= lo[1]) & (j <= hi[1])
                    mk = (k >= lo[2]) & (k <= hi[2])
                    if not (mi.any() and mj.any() and mk.any()) or px >= cfg.npix_x or py >= cfg.npix_y:
                        continue
                    key = (int(bt[b]) * cfg.npix_x + int(px)) * cfg.npix_y + int(py)
                    acc[key] = acc.get(key, 0.0) + float(pay[b][np.ix_(mi, mj, mk)].sum())
        for key in sorted(acc):
            rs.append(s); rk.append(key); rq.append(acc[key])
    return np.asarray(rs, np.int32), np.asarray(rk, np.int64), np.asarray(rq, np.float64)
