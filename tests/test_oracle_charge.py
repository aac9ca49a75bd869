"""Pins of the oracle's quadrature constants, charge density (Eq. 10) and effective
charge (Eq. 9) against what the paper and the mathematics fix -- not against the
oracle itself.  CPU only."""
import os

import numpy as np
import pytest
from scipy import integrate, interpolate, special

import gen
import oracle as o

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden_gl():
    rows = {}
    for line in open(os.path.join(GOLD, "gauss_legendre.txt")):
        line = line.split("#")[0].split()
        if len(line) == 3:
            rows.setdefault(int(line[0]), []).append((float(line[1]), float(line[2])))
    return rows


# --------------------------------------------------------------------------- GL rule
@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_gl_matches_textbook_values(n):
    """PAPER.md:L85-89; tests/golden/gauss_legendre.txt holds the closed forms."""
    xi, w = o.gl_rule(n)
    ref = np.array(_golden_gl()[n])
    np.testing.assert_allclose(xi, ref[:, 0], atol=1e-15)
    np.testing.assert_allclose(w, ref[:, 1], atol=1e-15)


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_gl_exact_to_degree_2n_minus_1(n):
    xi, w = o.gl_rule(n)
    assert abs(w.sum() - 2.0) < 1e-15
    for deg in range(2 * n):
        exact = 0.0 if deg % 2 else 2.0 / (deg + 1)
        assert abs(np.sum(w * xi ** deg) - exact) < 1e-14
    # and NOT exact at degree 2n (so the test would notice a higher-order rule)
    assert abs(np.sum(w * xi ** (2 * n)) - 2.0 / (2 * n + 1)) > 1e-4


# --------------------------------------------------------------------------- u table
@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_trilinear_u_partition_of_unity_and_linear_reproduction(n):
    """Eq. (7): the 1-D factors interpolate linearly between cuboid centres, so they
    sum to 1 and reproduce the node position  sum_r u_r (c + r) = c + xi/2."""
    xi, _ = o.gl_rule(n)
    u = o.trilinear_u(xi)
    np.testing.assert_allclose(u.sum(1), 1.0, atol=1e-15)
    np.testing.assert_allclose(u @ np.array([-1.0, 0.0, 1.0]), xi / 2, atol=1e-15)
    assert (u >= 0).all()
    # a node left of the centre never touches the right neighbour and vice versa
    assert (u[xi < 0, 2] == 0).all() and (u[xi > 0, 0] == 0).all()


# --------------------------------------------------------------------------- Eq. (10)
def _aug1(p0, p1, sig, Q, flag=0):
    return dict(p0=np.array([p0], float), p1=np.array([p1], float), sig=np.array([sig], float),
                Qp=np.array([Q], float), flag=np.array([flag], np.int32))


def _line_gauss_quad(p0, p1, sig, Q, pos):
    """The DEFINITION: uniform line charge Q on [p0,p1] convolved with
    a 3-D Gaussian: q(x) = Q int_0^1 ds prod_a N(x_a; p0_a + s d_a, sig_a)."""
    p0, p1, sig, pos = map(np.asarray, (p0, p1, sig, pos))

    def f(s):
        m = p0 + s * (p1 - p0)
        return np.prod(np.exp(-0.5 * ((pos - m) / sig) ** 2) / (np.sqrt(2 * np.pi) * sig))
    return Q * integrate.quad(f, 0.0, 1.0, epsabs=0, epsrel=1e-13, limit=200)[0]


def test_eq10_equals_quadrature_of_its_definition():
    rng = np.random.default_rng(7)
    for _ in range(40):
        p0 = rng.uniform(-2, 2, 3)
        p1 = p0 + rng.uniform(-1.5, 1.5, 3)
        sig = rng.uniform(0.3, 1.5, 3)
        pos = 0.5 * (p0 + p1) + rng.normal(0, 1.0, 3) * sig
        Q = rng.uniform(1e3, 1e4)
        got = o.charge_density(_aug1(p0, p1, sig, Q), 0, pos)
        ref = _line_gauss_quad(p0, p1, sig, Q, pos)
        assert abs(got - ref) <= 1e-11 * abs(ref) + 1e-300


def test_eq10_in_the_papers_own_notation():
    """Eq. (10) with A_1, A_2, B, Delta^2 exactly as printed at PAPER.md:L135-140,
    except the exponent read as exp(-B / (2 Delta^2)) (reading G1).
    The printed exponent exp(-B/Delta^2) must NOT agree (guards the reading)."""
    rng = np.random.default_rng(8)
    worst_printed = 0.0
    for _ in range(20):
        (x0, y0, z0), (x1, y1, z1) = rng.uniform(-2, 2, 3), rng.uniform(-2, 2, 3)
        sx, sy, sz = rng.uniform(0.4, 1.2, 3)
        x, y, z = rng.uniform(-2, 2, 3)
        D2 = sy**2*sz**2*(x0-x1)**2 + sz**2*sx**2*(y0-y1)**2 + sx**2*sy**2*(z0-z1)**2
        A1 = sy**2*sz**2*(x-x0)*(x0-x1) + sz**2*sx**2*(y-y0)*(y0-y1) + sx**2*sy**2*(z-z0)*(z0-z1)
        A2 = sy**2*sz**2*(x-x1)*(x0-x1) + sz**2*sx**2*(y-y1)*(y0-y1) + sx**2*sy**2*(z-z1)*(z0-z1)
        B = (sy**2*(x*(z0-z1) + (z1*x0-z0*x1) - z*(x0-x1))**2
             + sz**2*(y*(x0-x1) + (x1*y0-x0*y1) - x*(y0-y1))**2
             + sx**2*(y*(z0-z1) + (z1*y0-z0*y1) - z*(y0-y1))**2)
        D = np.sqrt(D2)
        er = special.erf(A2/(np.sqrt(2)*D*sx*sy*sz)) - special.erf(A1/(np.sqrt(2)*D*sx*sy*sz))
        Q = 5000.0
        corrected = Q*np.exp(-B/(2*D2))/(4*np.pi*D)*er
        printed = Q*np.exp(-B/D2)/(4*np.pi*D)*er
        got = o.charge_density(_aug1((x0, y0, z0), (x1, y1, z1), (sx, sy, sz), Q), 0, (x, y, z))
        ref = _line_gauss_quad((x0, y0, z0), (x1, y1, z1), (sx, sy, sz), Q, (x, y, z))
        assert abs(got - corrected) <= 1e-10 * abs(corrected)
        assert abs(corrected - ref) <= 1e-10 * abs(ref)
        worst_printed = max(worst_printed, abs(printed - ref) / abs(ref))
    assert worst_printed > 0.1


def test_eq10_swap_invariance_and_point_limit():
    rng = np.random.default_rng(9)
    for _ in range(10):
        p0 = rng.uniform(-1, 1, 3); p1 = p0 + rng.uniform(-1, 1, 3)
        sig = rng.uniform(0.3, 1.0, 3); pos = rng.uniform(-1.5, 1.5, 3)
        a = o.charge_density(_aug1(p0, p1, sig, 1e4), 0, pos)
        b = o.charge_density(_aug1(p1, p0, sig, 1e4), 0, pos)
        assert abs(a - b) <= 1e-12 * abs(a)
    # short-segment limit: line form -> point Gaussian at the midpoint
    p0 = np.array([0.3, -0.2, 0.1]); d = np.array([1e-4, -2e-4, 1.5e-4]); sig = np.array([0.5, 0.6, 0.7])
    pos = np.array([0.6, 0.1, -0.3])
    line = o.charge_density(_aug1(p0, p0 + d, sig, 1e4, 0), 0, pos)
    point = o.charge_density(_aug1(p0, p0 + d, sig, 1e4, 1), 0, pos)
    mid = p0 + 0.5 * d
    closed = 1e4 * np.prod(np.exp(-0.5*((pos-mid)/sig)**2) / (np.sqrt(2*np.pi)*sig))
    assert abs(point - closed) <= 1e-13 * closed
    assert abs(line - point) <= 1e-6 * point


# --------------------------------------------------------------------------- Eq. (9)
def _tiny_cfg(n, nsigma=4.0, **kw):
    base = dict(npix_x=4, npix_y=4, nticks=96, gl_n=n, block=(8, 8, 32), resp_nticks=16,
                nsigma=nsigma, t_origin_us=0.0)
    base.update(kw)
    return gen.make_config(1, **base)


def _one_seg(cfg, z=160.0, d=(0.6, -0.5, 0.7), q=6000.0, centre=None):
    """One segment whose charge cloud sits inside the 4x4-pixel, 96-tick window."""
    cx = cfg.npix_x * cfg.pitch_mm / 2 if centre is None else centre[0]
    cy = cfg.npix_y * cfg.pitch_mm / 2 if centre is None else centre[1]
    p0 = np.array([cx, cy, z]) - 0.5 * np.array(d)
    p1 = p0 + np.array(d)
    s = dict(x0=p0[0], y0=p0[1], z0=p0[2], x1=p1[0], y1=p1[1], z1=p1[2], q=q, t0=0.0)
    return {k: np.array([v], np.float32) for k, v in s.items()}


def _dense_effq(cfg, segs):
    aug = o.drift(cfg, segs)
    keys = o.blocks(cfg, aug)
    return aug, keys, o.payload_to_dense(cfg, keys, o.effq(cfg, aug, keys))


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_total_effective_charge_equals_attenuated_charge(n):
    """north_star: total effective charge = deposited charge x exp(-t_drift/tau).
    With sigma >= h and a 6-sigma box the quadrature + truncation error is < 1e-7
    (SURVEY.md Sec. 8(c) G8); n=1 is the midpoint rule (looser)."""
    z = 160.0                                   # t_m = 100 us -> sigma_T = 0.49 mm > h = 0.44
    cfg = _tiny_cfg(n, nsigma=6.0, t_origin_us=z / 1.6 - 4.8)
    segs = _one_seg(cfg, z=z)
    aug, keys, dense = _dense_effq(cfg, segs)
    expect = 6000.0 * np.exp(-(z / 1.6) / 2200.0)
    assert abs(aug["Qp"][0] - expect) < 1e-9 * expect
    tol = {1: 2e-3, 2: 1e-4, 3: 3e-6, 4: 2e-7}[n]
    assert abs(dense.sum() - expect) < tol * expect


def test_n1_is_sampling_at_grid_points():
    """PAPER.md:L274-276 calls the 1-point rule "sampling at grid points":
    Qeff[i,j,k] = hx hy ht q(grid point) with the grid point at the cuboid centre."""
    z = 160.0
    cfg = _tiny_cfg(1, t_origin_us=z / 1.6 - 4.8)
    segs = _one_seg(cfg, z=z)
    aug, keys, dense = _dense_effq(cfg, segs)
    g = o.grid_of(cfg)
    lo, hi = aug["lo"][0], aug["hi"][0]
    rng = np.random.default_rng(3)
    vol = g.h[0] * g.h[1] * g.h[2]
    for _ in range(50):
        ijk = [int(rng.integers(lo[a], hi[a] + 1)) for a in range(3)]
        pos = [g.org[a] + (ijk[a] + 0.5) * g.h[a] for a in range(3)]
        ref = vol * o.charge_density(aug, 0, pos)
        assert abs(dense[tuple(ijk)] - ref) <= 1e-13 * abs(ref) + 1e-30
    assert dense[lo[0] - 1 if lo[0] > 0 else 0, :, :].sum() == 0 or lo[0] == 0


@pytest.mark.parametrize("n", [2, 3, 4])
def test_eq9_adjoint_identity_with_independent_trilinear_interpolation(n):
    """Eq. (4)-(9): sum_g Qeff[g] I[g] must equal sum_nodes w q(node) I_interp(node),
    with I_interp the piecewise-trilinear interpolant of the grid function I through
    the cuboid CENTRES.  The right-hand side is computed here with scipy's
    RegularGridInterpolator and an explicit loop over nodes -- no oracle scatter code."""
    z = 120.0
    cfg = _tiny_cfg(n, nsigma=3.0, t_origin_us=z / 1.6 - 3.0, nticks=64)
    segs = _one_seg(cfg, z=z, d=(0.9, 0.4, -0.6))
    aug, keys, dense = _dense_effq(cfg, segs)
    g = o.grid_of(cfg)
    rng = np.random.default_rng(11)
    I = rng.standard_normal(dense.shape)
    axes = [g.org[a] + (np.arange(g.NG[a]) + 0.5) * g.h[a] for a in range(3)]
    interp = interpolate.RegularGridInterpolator(axes, I, method="linear")
    xi, w = o.gl_rule(n)
    lo, hi = aug["lo"][0], aug["hi"][0]
    assert (lo >= 1).all() and all(hi[a] < g.NG[a] - 1 for a in range(3))   # fully inside
    rhs = 0.0
    for cx in range(lo[0], hi[0] + 1):
        for cy in range(lo[1], hi[1] + 1):
            for ct in range(lo[2], hi[2] + 1):
                for l in range(n):
                    for m in range(n):
                        for k in range(n):
                            pos = (g.org[0] + (cx + 0.5 + 0.5 * xi[l]) * g.h[0],
                                   g.org[1] + (cy + 0.5 + 0.5 * xi[m]) * g.h[1],
                                   g.org[2] + (ct + 0.5 + 0.5 * xi[k]) * g.h[2])
                            wt = w[l] * w[m] * w[k] * g.h[0] * g.h[1] * g.h[2] / 8.0
                            rhs += wt * o.charge_density(aug, 0, pos) * float(interp(np.array([pos]))[0])
    lhs = float((dense * I).sum())
    assert abs(lhs - rhs) <= 1e-10 * np.abs(dense).sum()


def test_effq_conserves_centroid_of_node_charges():
    """u reproduces linear functions, so sum_g Qeff[g] x_g equals the GL quadrature of
    int q x dV; with sigma >= h and 6 sigma that is Q' x (segment midpoint)."""
    z = 160.0
    cfg = _tiny_cfg(3, nsigma=6.0, t_origin_us=z / 1.6 - 4.8)
    segs = _one_seg(cfg, z=z)
    aug, keys, dense = _dense_effq(cfg, segs)
    g = o.grid_of(cfg)
    mid = 0.5 * (aug["p0"][0] + aug["p1"][0])
    for a in range(3):
        x = g.org[a] + (np.arange(g.NG[a]) + 0.5) * g.h[a]
        shape = [1, 1, 1]; shape[a] = -1
        cen = (dense * x.reshape(shape)).sum() / dense.sum()
        assert abs(cen - mid[a]) < 2e-5 * g.h[a]


def test_effq_linearity_and_translation_equivariance():
    """north_star: charge linearity; translation by one whole pixel / one tick shifts
    Qeff by exactly S grid points / one tick."""
    z = 100.0
    cfg = _tiny_cfg(2, t_origin_us=z / 1.6 - 3.0, npix_x=6, npix_y=6)
    c0 = (2.5 * cfg.pitch_mm + 0.3, 2.5 * cfg.pitch_mm - 0.4)
    a = _dense_effq(cfg, _one_seg(cfg, z=z, q=5000.0, centre=c0))[2]
    b = _dense_effq(cfg, _one_seg(cfg, z=z, q=10000.0, centre=c0))[2]
    np.testing.assert_allclose(b, 2 * a, rtol=1e-6, atol=1e-9)    # q is fp32 on input
    c1 = (c0[0] + cfg.pitch_mm, c0[1] - cfg.pitch_mm)
    s = _dense_effq(cfg, _one_seg(cfg, z=z, q=5000.0, centre=c1))[2]
    S = cfg.sub
    ref = np.zeros_like(a); ref[S:, :-S, :] = a[:-S, S:, :]
    # fp32 input coordinates differ by rounding of the shift -> compare loosely
    assert np.abs(s - ref).max() < 2e-4 * np.abs(a).max()
    # exact tick shift through t_origin (no input rounding involved)
    cfg2 = cfg.with_(t_origin_us=cfg.t_origin_us - cfg.tick_us * 3)
    t = _dense_effq(cfg2, _one_seg(cfg2, z=z, q=5000.0, centre=c0))[2]
    ref = np.zeros_like(a); ref[:, :, 3:] = a[:, :, :-3]
    assert np.abs(t - ref).max() < 1e-7 * np.abs(a).max()


def test_fig7_ordering_of_quadrature_error():
    """PAPER.md:L276-278 (Fig. 7): relative to the 4-point rule, sampling at grid
    points (n=1) deviates clearly more than the 2-point rule.  Only the ORDERING is
    pinned (their response and data are unavailable: magnitudes are parity-unpinned).
    Measured on the per-pixel, per-tick accumulated charge of one small-sigma segment."""
    z = 30.0                                     # sigma_T = 0.21 mm < h: hard case
    out = {}
    for n in (1, 2, 4):
        cfg = _tiny_cfg(n, t_origin_us=z / 1.6 - 3.0, sigma_min_xy_mm=0.05, sigma_min_t_us=0.01)
        dense = _dense_effq(cfg, _one_seg(cfg, z=z, d=(0.7, 0.6, 0.4)))[2]
        S = cfg.sub
        out[n] = dense.reshape(cfg.npix_x, S, cfg.npix_y, S, -1).sum((1, 3))
    e1 = np.sqrt(np.mean((out[1] - out[4]) ** 2))
    e2 = np.sqrt(np.mean((out[2] - out[4]) ** 2))
    assert e1 > 3.0 * e2 > 0
