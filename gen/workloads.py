"""Synthetic workloads standing in for the paper's GENIE -> edep-sim sample
(Sec. IV-A), which is not available.  Shapes follow
BASELINE.json `configs` 1..5; the recipe is restated in DESIGN.md.

Nothing here is TRED arithmetic: only seeded random geometry, a plain-data
configuration record and a seeded synthetic field response.
Units: mm, microseconds, electrons.
"""
from __future__ import annotations

from dataclasses import dataclass, replace, asdict
import numpy as np

SEG_FIELDS = ("x0", "y0", "z0", "x1", "y1", "z1", "q", "t0")


@dataclass(frozen=True)
class Config:
    """Plain-data record mirrored by `tred_config` in include/tred.h."""
    name: str
    npix_x: int
    npix_y: int
    nticks: int
    gl_n: int
    block: tuple            # (Bx, By, Bt) in fine-grid points / ticks
    resp_nticks: int
    sub: int = 10           # sub-pixel factor S (10x10 impact positions)
    resp_half: int = 5      # H: response covers (2H+1)^2 pixels
    pitch_mm: float = 4.4
    tick_us: float = 0.1
    origin_x_mm: float = 0.0
    origin_y_mm: float = 0.0
    t_origin_us: float = 0.0
    v_mm_us: float = 1.6
    lifetime_us: float = 2200.0
    DL_mm2_us: float = 7.2e-4       # 7.2 cm^2/s
    DT_mm2_us: float = 1.2e-3       # 12.0 cm^2/s
    sigma_min_xy_mm: float = 0.22   # h/2
    sigma_min_t_us: float = 0.05    # tick/2
    nsigma: float = 4.0
    point_thresh: float = 0.1
    drift_mm: float = 500.0         # generator only: depth of the drift volume
    effq_mode: int = 0              # tred_config.effq_mode (kernel variant, 0 = default)
    mac_mode: int = 0               # tred_config.mac_mode  (kernel variant, 0 = default)

    def with_(self, **kw) -> "Config":
        return replace(self, **kw)

    def as_dict(self) -> dict:
        return asdict(self)


_BASE = {
    1: dict(name="cfg1_single_track", npix_x=32, npix_y=32, nticks=1024, gl_n=2,
            block=(8, 8, 64), resp_nticks=200),
    2: dict(name="cfg2_neutrino_event", npix_x=128, npix_y=128, nticks=4096, gl_n=3,
            block=(8, 8, 64), resp_nticks=400, t_origin_us=-5.0),
    3: dict(name="cfg3_beam_spill", npix_x=230, npix_y=230, nticks=5000, gl_n=4,
            block=(16, 16, 128), resp_nticks=400, t_origin_us=-5.0),
    4: dict(name="cfg4_pileup", npix_x=700, npix_y=700, nticks=8000, gl_n=3,
            block=(16, 16, 128), resp_nticks=400, t_origin_us=-5.0),
}


def make_config(cfg_id: int, **overrides) -> Config:
    """Config 1..4 of BASELINE.json; config 5 = config 3 with `block`/`gl_n` overridden."""
    if cfg_id == 5:
        cfg_id = 3
    base = dict(_BASE[cfg_id])
    base.update(overrides)
    return Config(**base)


# ----------------------------------------------------------------------------
# track geometry
# ----------------------------------------------------------------------------
def _isotropic(rng, n):
    cz = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(1.0 - cz * cz)
    return np.stack([s * np.cos(ph), s * np.sin(ph), cz], axis=1)


def _split_track(start, direc, length, box, seg_len, reflect):
    """Cut the straight line start + s*direc, s in [0,length], every `seg_len`
    and (if `reflect`) at every crossing of a box face, folding it specularly
    back into the box.  Returns (p0[n,3], p1[n,3])."""
    cuts = [np.arange(0.0, length, seg_len), np.array([length])]
    if reflect:
        for a in range(3):
            d = direc[a]
            if abs(d) < 1e-12:
                continue
            e0, e1 = start[a], start[a] + d * length
            m_lo = int(np.floor(min(e0, e1) / box[a]))
            m_hi = int(np.ceil(max(e0, e1) / box[a]))
            ms = np.arange(m_lo, m_hi + 1)
            s = (ms * box[a] - start[a]) / d
            cuts.append(s[(s > 0.0) & (s < length)])
    s = np.unique(np.concatenate(cuts))
    s0, s1 = s[:-1], s[1:]
    keep = (s1 - s0) > 1e-6
    s0, s1 = s0[keep], s1[keep]
    p0 = start[None, :] + s0[:, None] * direc[None, :]
    p1 = start[None, :] + s1[:, None] * direc[None, :]
    if reflect:
        mid = 0.5 * (p0 + p1)
        for a in range(3):
            cell = np.floor(mid[:, a] / box[a])
            odd = (cell.astype(np.int64) & 1) == 1
            lo = cell * box[a]
            f0 = np.where(odd, (lo + box[a]) - p0[:, a], p0[:, a] - lo)
            f1 = np.where(odd, (lo + box[a]) - p1[:, a], p1[:, a] - lo)
            p0[:, a] = np.clip(f0, 0.0, box[a])
            p1[:, a] = np.clip(f1, 0.0, box[a])
    return p0, p1


def _pack(rng, p0_list, p1_list, t0_list, charge_per_mm=6000.0):
    p0 = np.concatenate(p0_list)
    p1 = np.concatenate(p1_list)
    t0 = np.concatenate(t0_list)
    ln = np.linalg.norm(p1 - p0, axis=1)
    q = charge_per_mm * ln * rng.uniform(0.8, 1.2, ln.shape[0])
    out = {
        "x0": p0[:, 0], "y0": p0[:, 1], "z0": p0[:, 2],
        "x1": p1[:, 0], "y1": p1[:, 1], "z1": p1[:, 2],
        "q": q, "t0": t0,
    }
    return {k: np.ascontiguousarray(v, dtype=np.float32) for k, v in out.items()}


def _event_tracks(rng, box, vertex, n_tracks, t0, p0s, p1s, t0s):
    dirs = _isotropic(rng, n_tracks)
    lens = np.exp(rng.uniform(np.log(50.0), np.log(1500.0), n_tracks))
    for d, L in zip(dirs, lens):
        a, b = _split_track(vertex, d, float(L), box, 1.0, True)
        p0s.append(a); p1s.append(b); t0s.append(np.full(a.shape[0], t0))


def _muon(rng, box, t0, p0s, p1s, t0s):
    pt = rng.uniform(0.0, 1.0, 3) * box
    d = _isotropic(rng, 1)[0]
    # extend both ways to the faces of the box
    with np.errstate(divide="ignore", invalid="ignore"):
        s_a = (0.0 - pt) / d
        s_b = (box - pt) / d
    s_hi = np.min(np.where(d != 0, np.maximum(s_a, s_b), np.inf))
    s_lo = np.max(np.where(d != 0, np.minimum(s_a, s_b), -np.inf))
    start = np.clip(pt + s_lo * d, 0.0, box)
    a, b = _split_track(start, d, float(s_hi - s_lo), box, 1.0, False)
    a = np.clip(a, 0.0, box); b = np.clip(b, 0.0, box)
    p0s.append(a); p1s.append(b); t0s.append(np.full(a.shape[0], t0))


def _spill(rng, box, n_vertices, t_offset, p0s, p1s, t0s, muons_per_vertex=5,
           tracks_lo=10, tracks_hi=60):
    for _ in range(n_vertices):
        vertex = rng.uniform(0.0, 1.0, 3) * box
        t0 = t_offset + rng.uniform(0.0, 10.0)
        n_tracks = int(rng.integers(tracks_lo, tracks_hi + 1))
        _event_tracks(rng, box, vertex, n_tracks, t0, p0s, p1s, t0s)
        for _ in range(muons_per_vertex):
            _muon(rng, box, t_offset + rng.uniform(0.0, 10.0), p0s, p1s, t0s)


def make_segments(cfg_id: int, seed: int | None = None, n_vertices: int | None = None,
                  n_spills: int | None = None):
    """Returns (Config, dict of float32 SoA arrays x0,y0,z0,x1,y1,z1,q,t0).

    z is the drift distance to the anode (mm), t0 the deposit time (us),
    q the ionisation electrons of the segment after recombination.
    `n_vertices` / `n_spills` shrink configs 3 / 4 for tests (same recipe)."""
    if cfg_id == 5:
        cfg_id = 3
    cfg = make_config(cfg_id)
    seed = 1000 + cfg_id if seed is None else seed
    rng = np.random.default_rng(seed)
    ext = np.array([cfg.npix_x * cfg.pitch_mm, cfg.npix_y * cfg.pitch_mm, cfg.drift_mm])
    p0s, p1s, t0s = [], [], []
    if cfg_id == 1:
        start = np.array([rng.uniform(0, ext[0]), rng.uniform(0, ext[1]), rng.uniform(50.0, 300.0)])
        d = _isotropic(rng, 1)[0]
        if start[2] + 300.0 * d[2] < 5.0:
            d[2] = -d[2]
        a, b = _split_track(start, d, 300.0, ext, 1.0, False)
        p0s.append(a); p1s.append(b); t0s.append(np.zeros(a.shape[0]))
        segs = _pack(rng, p0s, p1s, t0s)
        z_min = float(min(segs["z0"].min(), segs["z1"].min()))
        t_or = np.floor((z_min / cfg.v_mm_us - 2.0) * 10.0) / 10.0
        cfg = cfg.with_(t_origin_us=float(t_or))
        return cfg, segs
    if cfg_id == 2:
        vertex = rng.uniform(0.0, 1.0, 3) * ext
        _event_tracks(rng, ext, vertex, 40, 0.0, p0s, p1s, t0s)
    elif cfg_id == 3:
        _spill(rng, ext, 50 if n_vertices is None else n_vertices, 0.0, p0s, p1s, t0s)
    elif cfg_id == 4:
        for s in range(10 if n_spills is None else n_spills):
            srng = np.random.default_rng(seed + s)
            off = float(rng.uniform(0.0, 400.0))
            _spill(srng, ext, 50 if n_vertices is None else n_vertices, off, p0s, p1s, t0s)
    else:
        raise ValueError(f"unknown config {cfg_id}")
    return cfg, _pack(rng, p0s, p1s, t0s)


# ----------------------------------------------------------------------------
# synthetic field response
# ----------------------------------------------------------------------------
def make_response(cfg: Config, seed: int) -> np.ndarray:
    """Seeded synthetic field response R[jx][jy][kx][ky][tau], float32,
    shape (S, S, 2H+1, 2H+1, Tr).  (kx,ky) = output pixel minus the pixel that
    contains the charge, stored at index k+H; (jx,jy) = sub-pixel phase of the
    charge.  A bipolar pulse whose amplitude decays as exp(-r/(1.5 pitch)) plus,
    on the collecting pixel only, a unipolar pulse of unit integral:
    sum_tau R = 1 for kx=ky=0 and 0 elsewhere (in fp64, before the cast).
    A function of r only, so R_{-i}^{-j} = R_i^j."""
    S, H, Tr = cfg.sub, cfg.resp_half, cfg.resp_nticks
    rng = np.random.default_rng(seed)
    tau_c = Tr * rng.uniform(0.70, 0.80)
    w = Tr * rng.uniform(0.04, 0.06)
    tau = np.arange(Tr, dtype=np.float64)
    bip = -(tau - tau_c) / w * np.exp(-0.5 * ((tau - tau_c) / w) ** 2)
    bip -= bip.mean()
    bip /= np.abs(bip).max()
    uni = np.exp(-0.5 * ((tau - tau_c - w) / (0.5 * w)) ** 2)
    uni /= uni.sum()
    h = cfg.pitch_mm / S
    j = np.arange(S, dtype=np.float64) + 0.5 - S / 2.0
    k = np.arange(-H, H + 1, dtype=np.float64)
    u = j[:, None] - S * k[None, :]                       # [S, 2H+1]
    r = h * np.sqrt(u[:, None, :, None] ** 2 + u[None, :, None, :] ** 2)   # [S,S,K,K]
    amp = uni.max() * np.exp(-r / (1.5 * cfg.pitch_mm))
    R = amp[..., None] * bip
    R[:, :, H, H, :] += uni
    return np.ascontiguousarray(R, dtype=np.float32)


def make_random_response(cfg: Config, seed: int) -> np.ndarray:
    """Unstructured (asymmetric) response for tests that pin index order and sign."""
    S, H, Tr = cfg.sub, cfg.resp_half, cfg.resp_nticks
    rng = np.random.default_rng(seed)
    K = 2 * H + 1
    return rng.standard_normal((S, S, K, K, Tr)).astype(np.float32)


# ----------------------------------------------------------------------------
# synthetic G4Steps (input of the step preprocessing): straight tracks cut
# into steps of random length (exponential, mean 4 mm, up to 40 mm), energy loss per unit
# length 2.1 MeV/cm x U(0.8, 3).  Geometry and energies only -- no arithmetic of the method.
# ----------------------------------------------------------------------------
STEP_FIELDS = ("x0", "y0", "z0", "x1", "y1", "z1", "dE", "t0")

STEP_PARAMS = dict(max_len_mm=5.0, recomb_model=1, w_ion_ev=23.6, efield_kv_cm=0.5, density_g_cm3=1.39,
                   birks_A=0.8, birks_k=0.0486, box_alpha=0.93, box_beta=0.212)


def make_steps(seed: int, n_tracks: int = 20, box_mm=(563.2, 563.2, 500.0)):
    rng = np.random.default_rng(seed)
    box = np.asarray(box_mm, dtype=np.float64)
    rows = []
    for _ in range(n_tracks):
        p = rng.uniform(0.0, 1.0, 3) * box
        d = _isotropic(rng, 1)[0]
        t0 = rng.uniform(0.0, 10.0)
        total = float(np.exp(rng.uniform(np.log(50.0), np.log(1500.0))))
        done = 0.0
        while done < total:
            ln = float(min(max(rng.exponential(4.0), 0.05), 40.0))
            q = p + ln * d
            if np.any(q < 0.0) or np.any(q > box):
                break
            dedx = 2.1 * rng.uniform(0.8, 3.0)                  # MeV/cm
            rows.append((*p, *q, dedx * ln / 10.0, t0))
            p = q
            done += ln
    a = np.asarray(rows, dtype=np.float32)
    return {k: np.ascontiguousarray(a[:, i]) for i, k in enumerate(STEP_FIELDS)}
