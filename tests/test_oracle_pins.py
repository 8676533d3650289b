"""Pins of the CPU oracle (oracle/dt_oracle.c) against things other than itself.

P1-P10 of SURVEY.md section 8(c) / DESIGN.md "Pins".  The paper prints no worked example and no
formula for any step (PAPER.md:141-143, 202 give the skeleton only), so the pins are: 40-digit
values of the definition (tests/golden, written by make_golden_mp.py, vector-form projection and a
different Kepler iteration), closed forms, invariants, an independent bisection solver, brute force
in numpy and injected-source statistics (BASELINE.json north_star lists exactly these four checks).
All CPU; none of this touches the CUDA package.
"""
import math

import numpy as np
import pytest

import dtsynth as ds
import oracle
from conftest import read_golden

K = ds.GAUSS_K
GM, C, EPS, S = ds.GM_SUN, ds.C_AU_PER_DAY, ds.OBLIQUITY, ds.PIXEL_SCALE
TWO_PI = 2.0 * math.pi


def survey(t, ra0, dec0, W=256, H=256, obs=None, c=C, var=None, mode=0):
    t = np.atleast_1d(np.asarray(t, float))
    obs = ds.observer_ecliptic(t) if obs is None else np.asarray(obs, float).reshape(-1, 3)
    return oracle.Survey(t, obs, np.atleast_1d(ra0), np.atleast_1d(dec0), W, H, S, GM, c, EPS, mode,
                         var)


# ---- P1 / P2: Kepler ------------------------------------------------------------------------------
def test_p1_kepler_residual_below_1e14():
    r = np.random.default_rng(1)
    worst = 0.0
    for e, M in zip(r.uniform(0, 0.97, 4000), r.uniform(-25, 25, 4000)):
        E, it, res = oracle.kepler(e, M)
        worst = max(worst, res)
        assert it < 50
    assert worst < 1e-14                      # north_star: "residuals below 1e-14"


def test_p2_kepler_values_40_digit():
    with open(__file__.replace("test_oracle_pins.py", "golden/kepler_values.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    assert len(rows) >= 10
    for e, M, E in rows:
        got, _, _ = oracle.kepler(float(e), float(M))
        # conditioning: dE = dM / (1 - e cos E); allow a few ulp of M through it
        cond = 1.0 / (1.0 - float(e) * math.cos(float(E)))
        diff = (got - float(E)) - TWO_PI * round((got - float(E)) / TWO_PI)   # E = +-pi are one point
        assert abs(diff) <= 4e-16 * max(1.0, cond) * max(1.0, abs(float(E))), (e, M)


def _bisect(e, m):
    lo, hi = 0.0, math.pi          # m in [0, pi]: root in [0, pi]
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if mid - e * math.sin(mid) < m:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def test_p2_kepler_vs_bisection():
    r = np.random.default_rng(2)
    for e, m in zip(r.uniform(0, 0.95, 500), r.uniform(0, math.pi, 500)):
        E, _, _ = oracle.kepler(e, m)
        Eb = _bisect(e, m)
        assert abs(E - Eb) <= 1e-15 * 4 / (1 - e) + 4e-16
        En, _, _ = oracle.kepler(e, -m)           # odd symmetry
        assert En == -E
        Ew, _, _ = oracle.kepler(e, m + 3 * TWO_PI)   # principal value returned
        assert abs(Ew - E) < 1e-13


def test_kepler_rejects_invalid():
    for e, M in [(1.0, 0.3), (-0.1, 0.3), (0.5, float("nan")), (0.5, float("inf"))]:
        with pytest.raises(ValueError):
            oracle.kepler(e, M)


# ---- P3 / P4: position ------------------------------------------------------------------------------
def test_p3_circular_closed_form():
    r = np.random.default_rng(3)
    for _ in range(200):
        a, inc = r.uniform(0.8, 40), r.uniform(0, 1.2)
        node, peri, M0 = r.uniform(0, TWO_PI, 3)
        t, t0 = r.uniform(-500, 500), r.uniform(-10, 10)
        pos, M, E = oracle.helio([a, 0.0, inc, node, peri, M0], GM, t, t0)
        n = math.sqrt(GM / a ** 3)
        u = peri + M0 + n * (t - t0)              # uniform mean motion (north_star)
        x, y, z = a * math.cos(u), a * math.sin(u) * math.cos(inc), a * math.sin(u) * math.sin(inc)
        want = [x * math.cos(node) - y * math.sin(node), x * math.sin(node) + y * math.cos(node), z]
        assert np.allclose(pos, want, rtol=0, atol=2e-13 * a * max(1.0, abs(u)))
        Ered = M - TWO_PI * round(M / TWO_PI)
        assert abs(E - Ered) < 1e-15 * max(1, abs(M))
    # i = 0: r = a (cos th, sin th, 0), th = Omega + omega + M
    pos, M, _ = oracle.helio([2.5, 0.0, 0.0, 0.7, 1.1, 0.3], GM, 100.0, 0.0)
    th = 0.7 + 1.1 + M
    assert np.allclose(pos, [2.5 * math.cos(th), 2.5 * math.sin(th), 0.0], atol=1e-14)


def test_p4_invariants():
    r = np.random.default_rng(4)
    for _ in range(200):
        a, e, inc = r.uniform(0.8, 40), r.uniform(0, 0.9), r.uniform(0, 1.2)
        node, peri, M0 = r.uniform(0, TWO_PI, 3)
        el = [a, e, inc, node, peri, M0]
        P, Q = oracle.pq(inc, node, peri)
        assert abs(P @ P - 1) < 1e-15 and abs(Q @ Q - 1) < 1e-15 and abs(P @ Q) < 1e-15
        h_hat = np.cross(P, Q)                    # orbit normal
        assert np.allclose(h_hat, [math.sin(inc) * math.sin(node), -math.sin(inc) * math.cos(node),
                                   math.cos(inc)], atol=1e-15)
        t = r.uniform(-1000, 1000)
        pos, M, E = oracle.helio(el, GM, t, 0.0)
        assert abs(np.linalg.norm(pos) - a * (1 - e * math.cos(E))) < 1e-14 * a
        assert abs(pos @ h_hat) < 1e-14 * a       # stays in the orbital plane
        # angular momentum and vis-viva by central finite difference
        n = math.sqrt(GM / a ** 3)
        dt = 1e-4 / n
        p1, _, _ = oracle.helio(el, GM, t + dt, 0.0)
        p0, _, _ = oracle.helio(el, GM, t - dt, 0.0)
        v = (p1 - p0) / (2 * dt)
        h = np.cross(pos, v)
        assert np.allclose(h, math.sqrt(GM * a * (1 - e * e)) * h_hat, rtol=0,
                           atol=1e-6 * np.linalg.norm(h))
        rn = np.linalg.norm(pos)
        assert abs(v @ v - GM * (2 / rn - 1 / a)) < 2e-6 * (v @ v)
    # perihelion at M = 0 along P, aphelion at M = pi along -P
    P, Q = oracle.pq(0.3, 1.0, 2.0)
    pos, _, _ = oracle.helio([3.0, 0.25, 0.3, 1.0, 2.0, 0.0], GM, 0.0, 0.0)
    assert np.allclose(pos, 3.0 * 0.75 * P, atol=1e-15)
    pos, _, _ = oracle.helio([3.0, 0.25, 0.3, 1.0, 2.0, math.pi], GM, 0.0, 0.0)
    assert np.allclose(pos, -3.0 * 1.25 * P, atol=1e-14)
    # quarter of the way in E: along Q with length b
    E = math.pi / 2
    pos, _, _ = oracle.helio([3.0, 0.25, 0.3, 1.0, 2.0, E - 0.25], GM, 0.0, 0.0)
    assert np.allclose(pos, -3.0 * 0.25 * P + 3.0 * math.sqrt(1 - 0.0625) * Q, atol=1e-14)


# ---- P5: light-time -----------------------------------------------------------------------------------
def test_p5_light_time_closed_form():
    # circular coplanar orbit: r(t - tau) is r(t) rotated by -n tau, tau = |r(t) - R| / c
    a, th0, t = 2.9, 1.3, 211.0
    el = [a, 0.0, 0.0, 0.0, 0.0, th0]
    sv = survey(t, 0.0, 0.0)
    p = oracle.pair(sv, el, 0.0, 0)
    n = math.sqrt(GM / a ** 3)
    th = th0 + n * t
    r = np.array([a * math.cos(th), a * math.sin(th), 0.0])
    R = ds.observer_ecliptic(np.array([t]))[0]
    tau = np.linalg.norm(r - R) / C
    assert abs(p.tau - tau) < 1e-15
    th1 = th - n * tau
    assert np.allclose(list(p.r1), [a * math.cos(th1), a * math.sin(th1), 0.0], atol=1e-14)
    assert 1e-3 < p.tau < 3e-2                      # ~ 8.3 min per AU
    # c = +inf: the geometric position
    pinf = oracle.pair(survey(t, 0.0, 0.0, c=float("inf")), el, 0.0, 0)
    assert pinf.tau == 0.0 and list(pinf.r1) == list(pinf.r)
    # exactly ONE iteration (A6): the converged light-time differs, and the oracle must not equal it
    tau2 = np.linalg.norm(np.array(list(p.r1)) - R) / C
    assert abs(tau2 - p.tau) > 1e-9


# ---- P6: frame + sky ------------------------------------------------------------------------------------
def test_p6_coplanar_sky_closed_form():
    r = np.random.default_rng(6)
    for _ in range(100):
        a, M0, t = r.uniform(1.5, 40), r.uniform(0, TWO_PI), r.uniform(0, 400)
        el = [a, 0.0, 0.0, 0.0, 0.0, M0]
        p = oracle.pair(survey(t, 0.0, 0.0), el, 0.0, 0)
        d = np.array(list(p.r1)) - ds.observer_ecliptic(np.array([t]))[0]
        lam = math.atan2(d[1], d[0])               # ecliptic longitude, latitude 0
        dec = math.asin(math.sin(EPS) * math.sin(lam))
        ra = math.atan2(math.cos(EPS) * math.sin(lam), math.cos(lam)) % TWO_PI
        assert abs(p.dec - dec) < 1e-15 and abs(p.ra - ra) < 2e-15
        assert abs(p.rho - np.linalg.norm(d)) < 1e-14 * a
    # sense of the rotation (A8): the ecliptic pole maps to dec = 90deg - eps at ra = 270deg
    t = 0.0
    obs = np.zeros((1, 3))
    sv = survey(t, 0.0, 0.0, obs=obs, c=float("inf"))
    # a polar orbit seen from the Sun at its northernmost point: i = 90deg, u = 90deg -> +z ecliptic
    p = oracle.pair(sv, [2.0, 0.0, math.pi / 2, 0.0, 0.0, math.pi / 2], 0.0, 0)
    assert abs(p.dec - (math.pi / 2 - EPS)) < 1e-15 and abs(p.ra - 1.5 * math.pi) < 1e-14


# ---- P7: gnomonic ---------------------------------------------------------------------------------------
def _sun_centred(ra, dec, rho=3.0):
    """Survey with the observer at the Sun, no light-time; returns elements of a circular orbit
    whose position at t = 0 has equatorial direction (ra, dec) -- built by inverse rotation."""
    q = np.array([math.cos(dec) * math.cos(ra), math.cos(dec) * math.sin(ra), math.sin(dec)])
    ce, se = math.cos(EPS), math.sin(EPS)
    d = np.array([q[0], q[1] * ce + q[2] * se, -q[1] * se + q[2] * ce])   # equatorial -> ecliptic
    lon, lat = math.atan2(d[1], d[0]), math.asin(d[2])
    # circular orbit with i = 90deg through that point: node = lon, argument of latitude = lat
    return [rho, 0.0, math.pi / 2, lon, 0.0, lat]


def test_p7_gnomonic_identities():
    r = np.random.default_rng(7)
    obs = np.zeros((1, 3))
    for _ in range(100):
        ra0, dec0 = r.uniform(0, TWO_PI), r.uniform(-1.2, 1.2)
        W, H = int(r.integers(16, 4096)), int(r.integers(16, 4096))
        sv = survey(0.0, ra0, dec0, W, H, obs=obs, c=float("inf"))
        # (i) object at the tangent point -> array centre
        p = oracle.pair(sv, _sun_centred(ra0, dec0), 0.0, 0)
        assert abs(p.x - (W - 1) / 2) < 1e-7 and abs(p.y - (H - 1) / 2) < 1e-7
        assert abs(p.D - 1) < 1e-15
        # (ii) inverse TAN of a pixel centre, re-projected -> same pixel (textbook inverse)
        ix, iy = int(r.integers(0, W)), int(r.integers(0, H))
        xi, eta = (ix - (W - 1) / 2) * S, (iy - (H - 1) / 2) * S
        den = math.cos(dec0) - eta * math.sin(dec0)
        ra = ra0 + math.atan2(xi, den)
        dec = math.atan2(math.sin(dec0) + eta * math.cos(dec0), math.hypot(xi, den))
        p = oracle.pair(sv, _sun_centred(ra, dec), 0.0, 0)
        assert (p.ix, p.iy) == (ix, iy) and p.hit == 1
        assert abs(p.x - ix) < 1e-6 and abs(p.y - iy) < 1e-6
        # (iii) trig form == vector form
        q = np.array(list(p.q))
        tv = np.array([math.cos(dec0) * math.cos(ra0), math.cos(dec0) * math.sin(ra0), math.sin(dec0)])
        ee = np.array([-math.sin(ra0), math.cos(ra0), 0.0])
        en = np.array([-math.sin(dec0) * math.cos(ra0), -math.sin(dec0) * math.sin(ra0), math.cos(dec0)])
        assert abs(p.xi - (q @ ee) / (q @ tv)) < 1e-15 and abs(p.eta - (q @ en) / (q @ tv)) < 1e-15
    # (iv) orientation (A9): +x east (increasing ra), +y north; small-angle limit xi -> dra cos(dec)
    sv = survey(0.0, 1.0, 0.5, 256, 256, obs=obs, c=float("inf"))
    pe = oracle.pair(sv, _sun_centred(1.0 + 2e-5, 0.5), 0.0, 0)
    pn = oracle.pair(sv, _sun_centred(1.0, 0.5 + 2e-5), 0.0, 0)
    assert abs(pe.xi - 2e-5 * math.cos(0.5)) < 1e-12 and abs(pe.eta) < 1e-9 and pe.x > 127.5
    assert abs(pn.eta - 2e-5) < 1e-12 and abs(pn.xi) < 1e-12 and pn.y > 127.5
    # (v) back hemisphere is culled (A10), footprint edges are half-open, rounding is floor(x + 1/2)
    pb = oracle.pair(sv, _sun_centred(1.0 + math.pi, -0.5), 0.0, 0)
    assert pb.D < 0 and pb.hit == 0 and (pb.ix, pb.iy) == (-1, -1)
    po = oracle.pair(sv, _sun_centred(1.0 + 200 * S / math.cos(0.5), 0.5), 0.0, 0)
    assert po.hit == 0 and po.x > 255.5
    for frac, want in [(0.49, 130), (0.51, 131), (-0.49, 130), (-0.51, 129)]:
        xi, eta = (130 + frac - 127.5) * S, 0.25 * S
        den = math.cos(0.5) - eta * math.sin(0.5)
        ph = oracle.pair(sv, _sun_centred(1.0 + math.atan2(xi, den),
                                          math.atan2(math.sin(0.5) + eta * math.cos(0.5),
                                                     math.hypot(xi, den))), 0.0, 0)
        assert (ph.ix, ph.iy) == (want, 128)


# ---- A11: the guard band (the tolerance of every GPU pixel comparison) ------------------------------------
def _place(ra0, dec0, W, H, xh, yh):
    """Elements of an object whose x + 1/2 = xh, y + 1/2 = yh on the tangent plane about (ra0, dec0):
    textbook inverse TAN, observer at the Sun, no light-time (independent of the oracle's forward chain)."""
    xi, eta = (xh - 0.5 - (W - 1) / 2) * S, (yh - 0.5 - (H - 1) / 2) * S
    den = math.cos(dec0) - eta * math.sin(dec0)
    ra = ra0 + math.atan2(xi, den)
    dec = math.atan2(math.sin(dec0) + eta * math.cos(dec0), math.hypot(xi, den))
    return _sun_centred(ra, dec)


def test_a11_guard_band_flag_is_1e6_px():
    """flag == 1 iff frac(x + 1/2) or frac(y + 1/2) lies within 1e-6 of 0 or 1 (reading A11, north_star:
    "within 1e-6 px of a rounding boundary").  Pairs are placed 5e-7 px (must flag) and 2e-6 px (must
    not) from a boundary, on either side, in x and in y, inside the image and at its four edges; the
    placement is checked to 1e-7 px on the oracle's own coordinate first, so a band of 1e-5 (or 1e-7)
    instead of 1e-6 fails here."""
    W, H = 256, 192
    ra0, dec0 = 1.0, 0.5
    sv = survey(0.0, ra0, dec0, W, H, obs=np.zeros((1, 3)), c=float("inf"))
    n_checked = 0
    for axis in (0, 1):
        size = W if axis == 0 else H
        for k in (0, 1, 57, size - 1, size):          # both footprint edges are rounding boundaries too
            for d, want in [(5e-7, 1), (-5e-7, 1), (2e-6, 0), (-2e-6, 0), (0.3, 0)]:
                other = 100.37                          # the other coordinate sits well inside a pixel
                xh, yh = (k + d, other) if axis == 0 else (other, k + d)
                p = oracle.pair(sv, _place(ra0, dec0, W, H, xh, yh), 0.0, 0)
                got = (p.x + 0.5, p.y + 0.5)
                assert abs(got[0] - xh) < 1e-7 and abs(got[1] - yh) < 1e-7, "placement"
                assert p.flag == want, (axis, k, d, p.flag)
                # the flag never changes the hit decision: half-open footprint, floor(x + 1/2)
                inside = 0.0 <= xh < W and 0.0 <= yh < H
                assert p.hit == int(inside)
                if inside:
                    assert (p.ix, p.iy) == (math.floor(xh), math.floor(yh))
                n_checked += 1
    assert n_checked == 50
    # both coordinates at once, and the project() array output carries the same flag
    els = [_place(ra0, dec0, W, H, 10 + 5e-7, 20 - 5e-7), _place(ra0, dec0, W, H, 10.5, 20.5)]
    out = oracle.project(sv, np.array(els), 0.0)
    assert out["flag"].tolist() == [[1], [0]]
    # behind the observer nothing is flagged
    pb = oracle.pair(sv, _sun_centred(ra0 + math.pi, -dec0), 0.0, 0)
    assert pb.D < 0 and pb.flag == 0


def test_a11_stack_counts_flagged_pairs_per_orbit():
    """dto_stack's nflag (what the GPU parity tests use to excuse an orbit): the number of the orbit's
    pairs that are flagged in or next to the footprint.  Scene: three exposures one day apart with the
    same tangent point on a 16384^2 image, observer at the Sun, no light-time; orbit A is placed 5e-7 px
    from a rounding boundary in exposure 0 and moves ~3400 px per day (unflagged, still inside, in
    exposures 1 and 2); orbit B sits 2e-6 px from the same boundary; orbit C is flagged but two pixels
    outside the footprint (not counted)."""
    W = H = 16384
    ra0, dec0 = 2.0, -0.3
    t = np.array([0.0, 1.0, 2.0])
    sv = oracle.Survey(t, np.zeros((3, 3)), np.full(3, ra0), np.full(3, dec0), W, H, S, GM, float("inf"), EPS,
                       0, np.ones(3))
    els = np.array([_place(ra0, dec0, W, H, 8000 + 5e-7, 8100.4),
                    _place(ra0, dec0, W, H, 8000 + 2e-6, 8100.4),
                    _place(ra0, dec0, W, H, -2.0 + 5e-7, 8100.4)])
    planes = [np.ones((H, W), np.float32)] * 3
    ref = oracle.stack(sv, planes, None, els, 0.0)
    flags = oracle.project(sv, els, 0.0)["flag"]
    assert flags[0, 0] == 1 and flags[1, 0] == 0 and flags[2, 0] == 1
    assert ref["hits"][0] == 3 and ref["hits"][1] == 3, ref["hits"]
    assert ref["nflag"].tolist() == [int(flags[0].sum()), int(flags[1].sum()), 0]
    assert ref["nflag"][0] == 1 and ref["nflag"][1] == 0
    assert abs(ref["snr"][0] - math.sqrt(3.0)) < 1e-15


# ---- P8: worked example --------------------------------------------------------------------------------
def test_p8_worked_example_we1():
    vals, consts = read_golden("we1.txt")
    assert consts["GM"] == GM and consts["c"] == C and consts["obliquity"] == EPS
    assert consts["pixel_scale"] == S
    el = [2.7, 0.1, math.radians(5), math.radians(80), math.radians(30), math.radians(250)]
    t = 17.25
    sv = survey(t, 6.0288, -0.2457, 256, 256, obs=[[math.cos(K * t), math.sin(K * t), 0.0]])
    p = oracle.pair(sv, el, 0.0, 0)
    got = dict(M=p.M, E=p.E - TWO_PI * round(p.E / TWO_PI), r_x=p.r[0], r_y=p.r[1], r_z=p.r[2],
               tau=p.tau, M1=p.M1, E1=p.E1 - TWO_PI * round(p.E1 / TWO_PI), r1_x=p.r1[0],
               r1_y=p.r1[1], r1_z=p.r1[2], q_x=p.q[0], q_y=p.q[1], q_z=p.q[2], rho=p.rho, ra=p.ra,
               dec=p.dec, D=p.D, xi=p.xi, eta=p.eta)
    for key, g in got.items():
        w = vals[key]
        if key in ("E", "E1"):
            w = w - TWO_PI * round(w / TWO_PI)
        assert abs(g - w) <= 4e-15 * max(1.0, abs(w)), key
    assert abs(p.x - vals["x"]) < 1e-8 and abs(p.y - vals["y"]) < 1e-8   # 1e-14 rad / 1e-6 rad/px
    assert (p.ix, p.iy, p.hit, p.flag) == (148, 79, 1, 0)
    assert p.kepler_resid < 1e-14


# ---- P9: stack -----------------------------------------------------------------------------------------
def _tiny_scene(n_orb=400, n_exp=24, W=64, H=64, mode=1, fraction=0.5):
    cfg = ds.focused(ds.scaled(ds.CONFIGS["tiny"], n_orbits=n_orb, n_exp=n_exp, width=W, height=H,
                               variance_mode=mode, var_range=(0.8, 1.2)), fraction=fraction)
    return ds.build_scene(cfg, oracle.scene_project_fn)


def test_p9_unit_images_give_sqrt_hits():
    sc = _tiny_scene()
    sv = oracle.Survey.from_scene(sc)
    N, (H, W) = sc.cfg.n_exp, (sc.cfg.height, sc.cfg.width)
    ones = [np.ones((H, W), np.float32)] * N
    out = oracle.stack(sv, ones, ones, sc.elements(), 0.0)
    assert out["hits"].max() >= N // 2 and (out["hits"] == 0).any()
    assert np.allclose(out["snr"], np.sqrt(out["hits"].astype(np.float64)), rtol=3e-16, atol=0)
    assert np.all(out["snr"][out["hits"] == 0] == 0.0)                          # A15


def test_p9_address_image_and_brute_force():
    sc = _tiny_scene()
    sv = oracle.Survey.from_scene(sc)
    N, (H, W) = sc.cfg.n_exp, (sc.cfg.height, sc.cfg.width)
    el = sc.elements()
    addr = [np.arange(H * W, dtype=np.float32).reshape(H, W) + 1000.0 * j for j in range(N)]
    var = [sc.var_plane_np(j) for j in range(N)]
    out = oracle.stack(sv, addr, var, el, 0.0)
    proj = oracle.project(sv, el, 0.0)
    # brute force in numpy from the per-pair pixels: gathered values ARE the pixel addresses
    pix = proj["pix"]
    for o in range(el.shape[0]):
        Ssum = Wsum = 0.0
        nh = 0
        for j in range(N):
            ix, iy = pix[o, j]
            if ix < 0:
                continue
            f = np.float64(np.float32(iy * W + ix + 1000.0 * j))
            v = np.float64(np.float32(sc.var_scalar[j]))
            Ssum += f / v
            Wsum += 1.0 / v
            nh += 1
        assert out["hits"][o] == nh
        assert out["S"][o] == Ssum and out["Wt"][o] == Wsum
        assert out["snr"][o] == (Ssum / math.sqrt(Wsum) if nh else 0.0)
    # scalar-variance mode reads var_scalar[j] (fp64) instead of the plane
    sc0 = _tiny_scene(mode=0)
    sv0 = oracle.Survey.from_scene(sc0)
    out0 = oracle.stack(sv0, addr, None, el, 0.0)
    o = int(np.argmax(out0["hits"]))
    js = np.flatnonzero(pix[o, :, 0] >= 0)
    want = sum(np.float64(addr[j][pix[o, j, 1], pix[o, j, 0]]) / sc0.var_scalar[j] for j in js)
    assert abs(out0["S"][o] - want) <= 1e-12 * abs(want)


def test_p9_masked_pixels_and_invalid_orbits():
    sc = _tiny_scene(n_orb=64)
    sv = oracle.Survey.from_scene(sc)
    N, (H, W) = sc.cfg.n_exp, (sc.cfg.height, sc.cfg.width)
    el = sc.elements()
    flux = [np.ones((H, W), np.float32) for _ in range(N)]
    var = [np.ones((H, W), np.float32) for _ in range(N)]
    base = oracle.stack(sv, flux, var, el, 0.0)
    o = int(np.argmax(base["hits"]))
    pix = oracle.project(sv, el[o:o + 1], 0.0)["pix"][0]
    js = np.flatnonzero(pix[:, 0] >= 0)
    flux[js[0]][pix[js[0], 1], pix[js[0], 0]] = np.nan          # A16: skipped, not counted
    var[js[1]][pix[js[1], 1], pix[js[1], 0]] = 0.0
    var[js[2]][pix[js[2], 1], pix[js[2], 0]] = np.inf
    out = oracle.stack(sv, flux, var, el, 0.0)
    assert out["hits"][o] == base["hits"][o] - 3
    assert abs(out["snr"][o] - math.sqrt(out["hits"][o])) < 1e-15 * 8
    bad = el.copy()
    bad[0, 0], bad[1, 1], bad[2, 1], bad[3, 5] = -1.0, 1.0, -0.1, np.nan
    outb = oracle.stack(sv, flux, var, bad, 0.0)
    assert list(outb["hits"][:4]) == [-1] * 4 and np.isnan(outb["snr"][:4]).all()
    assert np.array_equal(outb["snr"][4:], out["snr"][4:])


def test_p9_injected_source_recovery():
    # north_star: amplitude A into sigma = 1 noise along a known orbit stacks to A sqrt(N) +- 1
    cfg = ds.CONFIGS["tiny"]
    sc = ds.build_scene(cfg, oracle.scene_project_fn)
    sv = oracle.Survey.from_scene(sc)
    N = cfg.n_exp
    el = sc.elements()
    o = int(sc.inj_index[0])
    assert o == 5105 and np.allclose(el[o, :3], [2.7, 0.1, math.radians(5)])
    var = [sc.var_plane_np(j) for j in range(N)]
    flux = [sc.flux_plane_np(j) for j in range(N)]
    out = oracle.stack(sv, flux, var, el[o:o + 1], 0.0)
    assert out["hits"][0] == N                                   # tangent points track it
    assert abs(out["snr"][0] - 0.5 * math.sqrt(N)) < 4.0         # one draw: 4 sigma
    # many noise realisations (other seeds): mean A sqrt(N) +- 1/sqrt(n), sd 1
    pix = sc.inj_pix[0]
    off = pix[:, 1].astype(np.int64) * cfg.width + pix[:, 0]
    snrs = []
    for seed in range(1, 301):
        z = np.array([ds.rng.normal_np(seed, ds.rng.STREAM_NOISE_BASE + j,
                                       ds.rng.STREAM_NOISE_BASE2 + j, off[j:j + 1])[0]
                      for j in range(N)])
        snrs.append(np.sum(z + 0.5) / math.sqrt(N))
    snrs = np.array(snrs)
    assert abs(snrs.mean() - 0.5 * math.sqrt(N)) < 4 / math.sqrt(300)
    assert 0.85 < snrs.std() < 1.15
    # Fig. 4 shape: perturbing a by 1e-3 AU walks off the track -> noise
    full = oracle.stack(sv, flux, var, el, 0.0)
    pert = el[o:o + 1].copy()
    pert[0, 0] += 1e-3
    outp = oracle.stack(sv, flux, var, pert, 0.0)
    assert outp["snr"][0] < full["snr"][o] - 1.0 or outp["hits"][0] < N


# ---- P10: top-k -----------------------------------------------------------------------------------------
def test_p10_topk_equals_full_sort():
    r = np.random.default_rng(10)
    snr = np.round(r.normal(size=5000), 1)           # many ties
    hits = r.integers(-1, 6, 5000).astype(np.int32)
    snr[hits < 0] = np.nan
    for k, mh in [(10, 0), (100, 3), (5000, 1), (7000, 0), (0, 0)]:
        idx, val = oracle.topk(snr, hits, k, mh)
        ok = np.flatnonzero((hits >= mh) & np.isfinite(snr))
        order = ok[np.lexsort((ok, -snr[ok]))]       # snr descending, index ascending
        want = order[:k]
        assert np.array_equal(idx, want) and np.array_equal(val, snr[want])
