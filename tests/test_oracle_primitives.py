"""Pins of the oracle's primitives (SURVEY.md §8(c) O-1 ... O-4, O-11) against what the
mathematics fixes: survey vectors, atan2/closed forms in float64, brute force, invariants.
CPU only."""
import math
import os

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
SIGMA = float(np.float32(0.055 / math.sqrt(12.0)))


# ---------------------------------------------------------------- O-1 phi16
def _vectors():
    rows = []
    for line in open(os.path.join(HERE, "golden", "phi16_vectors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        x, y, p = line.split()
        rows.append((float(x), float(y), int(p)))
    return rows


def test_phi16_survey_vectors():
    rows = _vectors()
    assert len(rows) == 15
    got = oracle.phi16([r[0] for r in rows], [r[1] for r in rows])
    assert got.tolist() == [r[2] for r in rows]


def test_phi16_tracks_atan2():
    # |phi16 + 0.5 - atan2(y,x)*32768/pi| <= 0.52 (polynomial error 0.017 unit)
    rng = np.random.default_rng(7)
    x = rng.uniform(-45, 45, 20000).astype(np.float32)
    y = rng.uniform(-45, 45, 20000).astype(np.float32)
    p = oracle.phi16(x, y).astype(np.float64)
    ref = np.arctan2(y.astype(np.float64), x.astype(np.float64)) * 32768.0 / math.pi
    d = p + 0.5 - ref
    d = (d + 32768.0) % 65536.0 - 32768.0  # the cut at +-pi
    assert np.abs(d).max() <= 0.52


def test_phi16_monotone_on_circle():
    # walking a circle counter-clockwise from -pi, phi16 never decreases (a sign or octant slip would)
    a = np.linspace(-math.pi + 1e-4, math.pi - 1e-4, 200001)
    p = oracle.phi16((17.3 * np.cos(a)).astype(np.float32), (17.3 * np.sin(a)).astype(np.float32)).astype(np.int32)
    assert (np.diff(p) >= 0).all()
    assert p[0] <= -32766 and p[-1] >= 32766


def test_phi16_symmetries_and_scale():
    rng = np.random.default_rng(3)
    x = rng.uniform(0.1, 40, 2000).astype(np.float32)
    y = rng.uniform(0.1, 40, 2000).astype(np.float32)
    p = oracle.phi16(x, y).astype(np.int32)
    # power-of-two scaling leaves t = mn/mx bit-identical
    assert (oracle.phi16(4 * x, 4 * y) == p).all()
    # reflection y -> -y maps the bin [k, k+1) to [-k-1, -k): phi16 = -k-1 except on exact bin edges
    q = oracle.phi16(x, -y).astype(np.int32)
    assert ((q == -p - 1) | (q == -p)).all() and (q == -p - 1).mean() > 0.99


def test_phi16_grid_checksum_regression_and_fma_control():
    from tests.golden.make_phi16_checksum import fnv1a64, grid
    want = [l.strip() for l in open(os.path.join(HERE, "golden", "phi16_grid_checksum.txt")) if not l.startswith("#")][0]
    x, y = grid()
    got = "%016x" % fnv1a64(oracle.phi16(x, y).astype(np.uint16).astype("<u2").tobytes())
    assert got == want
    # negative control from SURVEY.md: an FMA-contracted evaluation gives a different checksum,
    # i.e. the grid is sensitive to contraction. Emulate FMA in float64 (exact product, one rounding).
    C = [np.float32(float.fromhex(h)) for h in ("0x1.fffd04p-1", "-0x1.549b14p-2", "0x1.8c5ee6p-3",
                                                "-0x1.dce202p-4", "0x1.af4978p-5", "-0x1.80032cp-7")]
    ax, ay = np.abs(x), np.abs(y)
    mx, mn = np.maximum(ax, ay), np.minimum(ax, ay)
    t = (mn / mx).astype(np.float32)
    s = (t * t).astype(np.float32)
    p = np.full_like(s, C[5])
    for c in (C[4], C[3], C[2], C[1], C[0]):
        p = (p.astype(np.float64) * s.astype(np.float64) + np.float64(c)).astype(np.float32)
    a = ((t * p).astype(np.float32) * np.float32(float.fromhex("0x1.45f306p+13"))).astype(np.float32)
    a = np.where(ay > ax, np.float32(16384.0) - a, a).astype(np.float32)
    a = np.where(x < 0, np.float32(32768.0) - a, a).astype(np.float32)
    a = np.where(y < 0, -a, a).astype(np.float32)
    k = np.floor(a).astype(np.int64)
    fma = (((k + 32768) & 65535) - 32768).astype(np.int16)
    assert "%016x" % fnv1a64(fma.astype(np.uint16).astype("<u2").tobytes()) != want


# ---------------------------------------------------------------- O-3 window
def test_window_matches_circular_distance_bruteforce():
    rng = np.random.default_rng(11)
    phis = np.concatenate([rng.integers(-32768, 32768, 300), [-32768, 32767, 0, -1, 1, 300, -300, 32468, -32468]])
    for W in (0, 1, 299, 300, 301, 5000, 32766, 32767, 32768, 40000, -1):
        for c in (-32768, -32600, -301, 0, 7, 32500, 32767):
            for p in phis:
                dist = min((int(p) - c) % 65536, (c - int(p)) % 65536)
                want = True if 2 * W + 1 >= 65536 else dist <= W
                assert oracle.in_window(int(p), c, W) == want, (p, c, W)


# ---------------------------------------------------------------- O-4 scatter
def test_scatter_hand_case_and_collinear():
    assert oracle.scatter((0, 0, 0), (1, 2, 10), (2, 5, 20)) == 1.0       # tz=1, ex=0, ey=-1
    assert oracle.scatter((0, 0, 0), (1, 2, 10), (2, 4, 20)) == 0.0       # exactly collinear
    assert oracle.scatter((1, -2, 100), (2, -4, 50), (4, -8, -50)) == 0.0  # unequal spacing, tz=2
    # a transposed operand or a sign error would change these
    assert oracle.scatter((0, 0, 0), (1, 0, 10), (3, 0, 20)) == 1.0
    assert oracle.scatter((0, 0, 0), (0, 1, 10), (0, 2, 30)) == 1.0       # predicted y=3, seen 2


def test_scatter_is_squared_extrapolation_miss_float64():
    rng = np.random.default_rng(5)
    for _ in range(2000):
        z = np.sort(rng.uniform(-300, 750, 3))[::-1]
        if min(z[0] - z[1], z[1] - z[2]) < 5:
            continue
        h = [(rng.uniform(-40, 40), rng.uniform(-40, 40), zz) for zz in z]
        h32 = [tuple(float(np.float32(v)) for v in p) for p in h]
        (x0, y0, z0), (x1, y1, z1), (x2, y2, z2) = h32
        px = x0 + (x1 - x0) * (z2 - z0) / (z1 - z0)
        py = y0 + (y1 - y0) * (z2 - z0) / (z1 - z0)
        want = (px - x2) ** 2 + (py - y2) ** 2
        got = oracle.scatter(*h32)
        assert abs(got - want) <= 1e-3 * want + 1e-6


# ---------------------------------------------------------------- O-2 sort
def test_sort_is_the_unique_total_order():
    rng = np.random.default_rng(9)
    n = 500
    # few distinct positions -> many equal (module, phi16) keys -> exercises the index tie-break
    px = rng.choice(np.array([-7.0, 3.5, 12.25, 0.0], np.float32), n)
    py = rng.choice(np.array([-2.0, 9.5, 0.0], np.float32), n)
    mod = rng.integers(0, 26, n).astype(np.uint8)
    mod[mod == 13] = 12   # an empty module in the middle
    perm, phi, mod_off = oracle.sort_event(px, py, mod, 26)
    assert sorted(perm.tolist()) == list(range(n))
    ph_all = oracle.phi16(px, py)
    keys = [(int(mod[i]), int(ph_all[i]), int(i)) for i in perm]
    assert keys == sorted((int(mod[i]), int(ph_all[i]), i) for i in range(n))
    assert (phi == ph_all[perm]).all()
    for m in range(27):
        assert mod_off[m] == int((mod < m).sum())
    assert mod_off[13] == mod_off[14] and mod_off[26] == n


def test_sort_empty_event():
    perm, phi, mod_off = oracle.sort_event(np.zeros(0, np.float32), np.zeros(0, np.float32), np.zeros(0, np.uint8), 26)
    assert perm.size == 0 and (mod_off == 0).all()


# ---------------------------------------------------------------- O-11 fit
def _fit64(hx, hy, hz, sigma):
    """Textbook simple linear regression in float64 (normal equations via numpy.polyfit), the
    point of closest approach of the fitted line to the z axis, and sigma^2 (A^T A)^-1 transported."""
    hx, hy, hz = (np.asarray(v, np.float64) for v in (hx, hy, hz))
    tx, cx = np.polyfit(hz, hx, 1)
    ty, cy = np.polyfit(hz, hy, 1)
    chi2 = (((hx - (cx + tx * hz)) ** 2).sum() + ((hy - (cy + ty * hz)) ** 2).sum()) / sigma ** 2
    s2 = tx * tx + ty * ty
    z = -(cx * tx + cy * ty) / s2 if s2 >= 1e-12 else hz.mean()
    A = np.stack([np.ones_like(hz), hz - z], axis=1)      # parameters (x at z, tx)
    cov = sigma ** 2 * np.linalg.inv(A.T @ A)
    return dict(x=cx + tx * z, y=cy + ty * z, tx=tx, ty=ty, z=z, chi2=chi2, cxx=cov[0, 0], cxtx=cov[0, 1], ctxtx=cov[1, 1])


def test_fit_matches_float64_regression():
    rng = np.random.default_rng(21)
    zs_all = np.array([1, 26, 51, 76, 101, 126, 151, 176, 201, 226, 251, 313, 390, 485, 604, 649, 694, 751], float)
    for _ in range(300):
        n = int(rng.integers(3, 15))
        i0 = int(rng.integers(0, len(zs_all) - n + 1))
        hz = zs_all[i0:i0 + n][::-1].copy()
        tx, ty = rng.uniform(-0.25, 0.25, 2)
        zv = rng.normal(0, 45)
        hx = tx * (hz - zv) + rng.normal(0, 0.016, n)
        hy = ty * (hz - zv) + rng.normal(0, 0.016, n)
        hx, hy, hz = (v.astype(np.float32) for v in (hx, hy, hz))
        o = oracle.fit(hx, hy, hz, SIGMA)
        w = _fit64(hx, hy, hz, SIGMA)
        assert abs(o[2] - w["tx"]) <= 1e-5 * abs(w["tx"]) + 1e-8
        assert abs(o[3] - w["ty"]) <= 1e-5 * abs(w["ty"]) + 1e-8
        if math.hypot(w["tx"], w["ty"]) > 0.01:
            # z = -(xb tx + yb ty)/s2 cancels: fp32 input rounding of ~1e-6 mm / slope
            assert abs(o[4] - w["z"]) <= 2e-5 * abs(w["z"]) + 2e-5 / math.hypot(w["tx"], w["ty"]) + 1e-3
            assert abs(o[0] - w["x"]) <= 1e-3 and abs(o[1] - w["y"]) <= 1e-3   # 1 um, SURVEY O-17
        assert abs(o[11] - w["chi2"]) <= 2e-3 * w["chi2"] + 1e-2
        for k, name in ((5, "cxx"), (6, "cxtx"), (7, "ctxtx")):
            assert abs(o[k] - w[name]) <= 1e-4 * abs(w[name]) + 1e-12, name
        assert o[8] == o[5] and o[9] == o[6] and o[10] == o[7]
        assert o[12:13].view(np.uint32)[0] == n


def test_fit_exact_collinear_and_line_through_axis():
    # SURVEY.md §8(c) whole-path pin (iii): x = 0.1 z, y = 0 at z = 51, 76, 101, 126
    hz = np.array([126, 101, 76, 51], np.float32)
    hx = (np.float32(0.1) * hz).astype(np.float32)
    o = oracle.fit(hx, np.zeros(4, np.float32), hz, SIGMA)
    assert abs(o[2] - 0.1) < 1e-6 and o[3] == 0.0
    assert abs(o[0]) < 1e-4 and o[1] == 0.0 and abs(o[4]) < 1e-3
    assert o[11] < 1e-3
    assert abs(o[7] - SIGMA ** 2 / 3125.0) <= 1e-6 * SIGMA ** 2 / 3125.0   # sdd = 2*(37.5^2+12.5^2)
    # exactly representable collinear points: slopes reproduced bit-exactly, chi2 == 0
    hz = np.array([100, 50, 0, -50], np.float32)
    o = oracle.fit(0.25 * hz + 2, -0.5 * hz - 4, hz, SIGMA)
    assert o[2] == 0.25 and o[3] == -0.5 and o[11] == 0.0
    # closest approach of (2+0.25z, -4-0.5z) to the z axis: z = -(2*0.25 + -4*-0.5)/(0.0625+0.25) = -8
    assert abs(o[4] + 8.0) < 1e-5 and abs(o[0] - 0.0) < 1e-5 and abs(o[1] - 0.0) < 1e-5
    # a line through (0, 0, z0=30): z = z0, x = y = 0
    hz = np.array([226, 201, 176], np.float32)
    o = oracle.fit(0.125 * (hz - 30), 0.0625 * (hz - 30), hz, SIGMA)
    assert abs(o[4] - 30.0) < 1e-4 and abs(o[0]) < 1e-5 and abs(o[1]) < 1e-5


def test_fit_degenerate_slope_A11():
    hz = np.array([76, 51, 26], np.float32)
    o = oracle.fit(np.full(3, 7.5, np.float32), np.full(3, -3.25, np.float32), hz, SIGMA)
    assert o[2] == 0 and o[3] == 0 and o[4] == 51.0 and o[0] == 7.5 and o[1] == -3.25 and o[6] == 0.0
