"""Pins of the oracle (oracle/opx_oracle.cpp) against things other than itself: known-answer
vectors, closed forms, textbook special cases, and an independent brute-force restatement in
NumPy fp64 with a *different* triangle test (Moeller-Trumbore).  CPU only.

P-numbers refer to SURVEY.md section 8(c) / DESIGN.md section 6.
"""
import os

import numpy as np
import pytest

import oracle
import workloads as wl
from workloads.photons import TrackSource, cherenkov_angle
from workloads.scenes import MAT_ABSORBER, MAT_DETECTOR, MAT_MIRROR, N_LAMBDA, Scene


def _golden(path):
    out = {}
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            k, v, tol = line.split()
            out[k] = (float(v), float(tol))
    return out


# ------------------------------------------------------------------------------------- P7 RNG
def test_p7_philox_known_answers(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        got = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in got] == v[6:10]


def test_p7_uniform_is_top_24_bits_of_word0():
    # ctr = (g lo, g hi, b, 0), key = (seed lo, seed hi); u = (word0 >> 8) * 2^-24
    assert oracle.uniform(0, 0, 0) == (0x6627e8d5 >> 8) * 2.0 ** -24
    assert abs(oracle.uniform(0, 0, 0) - 0.39904642) < 1e-8
    g, seed, b = 0x85a308d3243f6a88, 0x299f31d0a4093822, 0x13198a2e
    w0 = int(oracle.philox4x32_10([g & 0xffffffff, g >> 32, b, 0], [seed & 0xffffffff, seed >> 32])[0])
    assert oracle.uniform(seed, g, b) == (w0 >> 8) * 2.0 ** -24
    # (seed, id, bounce) each change the draw
    base = oracle.uniform(1, 2, 3)
    assert len({base, oracle.uniform(2, 2, 3), oracle.uniform(1, 3, 3), oracle.uniform(1, 2, 4),
                oracle.uniform(1, 2 + 2 ** 32, 3), oracle.uniform(1 + 2 ** 32, 2, 3)}) == 6


def test_p7_uniform_moments():
    u = np.array([oracle.uniform(7, g, 0) for g in range(20000)])
    assert 0.0 <= u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 4 * np.sqrt(1 / 12 / len(u))
    assert abs((u < 0.25).mean() - 0.25) < 4 * np.sqrt(0.25 * 0.75 / len(u))


# ------------------------------------------------------------------------------ P2 reflection
@pytest.mark.parametrize("fp64", [True, False])
def test_p2_law_of_reflection(fp64):
    rng = np.random.default_rng(1)
    tol = 1e-14 if fp64 else 4e-7
    for _ in range(200):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        n = rng.normal(size=3); n /= np.linalg.norm(n)
        if not fp64:
            d, n = d.astype(np.float32).astype(np.float64), n.astype(np.float32).astype(np.float64)
        r = oracle.reflect(d, n, fp64=fp64)
        assert abs(r @ n + d @ n) < tol                       # angle of incidence = angle of reflection
        assert abs(np.cross(d, n) @ r) < tol                  # r in the plane of d and n
        assert abs(np.linalg.norm(r) - np.linalg.norm(d)) < tol
        np.testing.assert_allclose(oracle.reflect(d, -n, fp64=fp64), r, atol=0, rtol=0)   # even in n
    # textbook case: 45 degrees off a plane with normal +z
    r = oracle.reflect([1 / np.sqrt(2), 0, -1 / np.sqrt(2)], [0, 0, 1], fp64=True)
    np.testing.assert_allclose(r, [1 / np.sqrt(2), 0, 1 / np.sqrt(2)], atol=1e-15)


def test_face_normal_is_unit_and_orthogonal():
    rng = np.random.default_rng(2)
    for _ in range(100):
        tri = rng.normal(size=(3, 3)).astype(np.float32) * 100
        n = oracle.face_normal(tri)
        t = tri.astype(np.float64)
        assert abs(np.linalg.norm(n) - 1) < 1e-14
        assert abs(n @ (t[1] - t[0])) < 1e-9 and abs(n @ (t[2] - t[0])) < 1e-9
        assert n @ np.cross(t[1] - t[0], t[2] - t[0]) > 0
    assert np.all(oracle.face_normal(np.zeros((3, 3))) == 0)   # degenerate triangle: zero normal


# ---------------------------------------------------------------------------- P10 table lookup
@pytest.mark.parametrize("fp64", [True, False])
def test_p10_table_lookup(fp64):
    rng = np.random.default_rng(3)
    y = rng.uniform(0, 1, N_LAMBDA).astype(np.float32)
    lam = 200.0 + 400.0 * np.arange(N_LAMBDA) / (N_LAMBDA - 1)
    for j in (0, 1, 17, 62, 63):
        if float(np.float32(lam[j])) == lam[j] or fp64:
            pass
        got = oracle.table_lerp(y, np.float32(lam[j]), fp64=fp64)
        assert abs(got - float(y[j])) < (1e-6 if not fp64 else 2e-6)   # float32 lambda is off the node by <= 1 ulp
    # exact nodes (200, 600 and every node that is an exact float): value returned exactly
    assert oracle.table_lerp(y, 200.0, fp64=fp64) == float(y[0])
    assert oracle.table_lerp(y, 600.0, fp64=fp64) == float(y[63])
    # clamped outside the grid, NaN-free
    assert oracle.table_lerp(y, 100.0, fp64=fp64) == float(y[0])
    assert oracle.table_lerp(y, 1e9, fp64=fp64) == float(y[63])
    # constant table returns the constant for every wavelength
    c = np.full(N_LAMBDA, 0.25, np.float32)
    for l in rng.uniform(150, 650, 50):
        assert oracle.table_lerp(c, l, fp64=fp64) == 0.25
    # linear table reproduces the line
    lin = (0.85 + 0.10 * np.arange(N_LAMBDA) / (N_LAMBDA - 1))
    for l in rng.uniform(200, 600, 200):
        l = float(np.float32(l))
        want = 0.85 + 0.10 * (l - 200.0) / 400.0
        assert abs(oracle.table_lerp(lin, l, fp64=fp64) - want) < (2e-7 if not fp64 else 4e-8)
    # piecewise linear between two nodes: midpoint of nodes 10, 11
    mid = float(np.float32(0.5 * (lam[10] + lam[11])))
    want = np.interp(mid, lam, y.astype(np.float64))
    assert abs(oracle.table_lerp(y, mid, fp64=fp64) - want) < 1e-5


# -------------------------------------------------------------------------------- P11 pixel map
@pytest.mark.parametrize("fp64", [True, False])
def test_p11_pixel_map(fp64):
    # axis-aligned frame with a pitch that is exact in binary so that edges are exact
    f = dict(A=np.float32([10, 20, 30]), u=np.float32([1, 0, 0]), v=np.float32([0, 0, 1]),
             pitch_u=0.5, pitch_v=0.25, nu=8, nv=4, pixel_base=0)
    for iu in range(8):
        for iv in range(4):
            ok, gu, gv = oracle.pixel_map(f, [10 + (iu + 0.5) * 0.5, 20, 30 + (iv + 0.5) * 0.25], fp64)
            assert ok and (gu, gv) == (iu, iv)                # pixel centres map to themselves
    assert oracle.pixel_map(f, [10 + 3 * 0.5, 99, 30 + 2 * 0.25], fp64) == (True, 3, 2)   # lower edges inclusive
    assert oracle.pixel_map(f, [10.0, 20, 30.0], fp64) == (True, 0, 0)                     # corner A itself
    assert oracle.pixel_map(f, [14.0, 20, 30.1], fp64)[0] is False                         # upper edge exclusive
    assert oracle.pixel_map(f, [10.1, 20, 31.0], fp64)[0] is False
    assert oracle.pixel_map(f, [9.999, 20, 30.1], fp64)[0] is False                        # negative a => outside
    assert oracle.pixel_map(f, [10.1, 20, 29.999], fp64)[0] is False
    # tilted frame of the toy RICH: pixel centres
    sc = wl.toy_rich_scene()
    fr, g = sc.frames[0], sc.info
    for iu, iv in [(0, 0), (207, 207), (104, 103), (81, 125)]:
        p = (fr["A"].astype(np.float64) + (iu + 0.5) * 2.88 * g["du"] + (iv + 0.5) * 2.88 * g["dv"])
        assert oracle.pixel_map(fr, p, fp64) == (True, iu, iv)


# ------------------------------------------------------------------------- ray/triangle test
def _moller_trumbore(o, d, tri):
    """Textbook Moeller-Trumbore in float64 (an independent formula)."""
    a, b, c = tri
    e1, e2 = b - a, c - a
    pv = np.cross(d, e2)
    det = e1 @ pv
    if det == 0:
        return None
    tv = o - a
    u = (tv @ pv) / det
    qv = np.cross(tv, e1)
    v = (d @ qv) / det
    if u < 0 or v < 0 or u + v > 1:
        return None
    return (e2 @ qv) / det, u, v


@pytest.mark.parametrize("fp64", [True, False])
def test_hit_triangle_matches_moller_trumbore(fp64):
    rng = np.random.default_rng(4)
    n_hit = 0
    for _ in range(3000):
        tri = (rng.normal(size=(3, 3)) * 50).astype(np.float32)
        o = (rng.normal(size=3) * 200).astype(np.float32)
        target = tri.astype(np.float64).T @ rng.dirichlet([1, 1, 1]) + rng.normal(size=3) * 20
        d = target - o
        d = (d / np.linalg.norm(d)).astype(np.float32)
        if rng.random() < 0.3:
            d = -d
        ref = _moller_trumbore(o.astype(np.float64), d.astype(np.float64), tri.astype(np.float64))
        hit, t = oracle.hit_triangle(o, d, tri, 0.0, fp64=fp64)
        if ref is not None and min(ref[1], ref[2], 1 - ref[1] - ref[2]) < 1e-4:
            continue                                          # too close to an edge to call in fp32
        want = ref is not None and ref[0] > 0
        assert hit == want
        if hit:
            n_hit += 1
            assert abs(t - ref[0]) < (1e-9 if fp64 else 2e-4) * max(1.0, abs(ref[0]))
    assert n_hit > 500


def test_hit_triangle_axis_cases_and_tmin():
    tri = np.float32([[-1, -1, 5], [3, -1, 5], [-1, 3, 5]])
    for fp64 in (True, False):
        assert oracle.hit_triangle([0, 0, 0], [0, 0, 1], tri, 0.0, fp64) == (True, 5.0)
        assert oracle.hit_triangle([0, 0, 10], [0, 0, -1], tri, 0.0, fp64) == (True, 5.0)   # no back-face culling
        assert oracle.hit_triangle([0, 0, 0], [0, 0, -1], tri, 0.0, fp64)[0] is False        # behind the origin
        assert oracle.hit_triangle([0, 0, 0], [0, 0, 1], tri, 5.0, fp64)[0] is False         # t > tmin is strict
        assert oracle.hit_triangle([0, 0, 5], [0, 0, 1], tri, 0.0, fp64)[0] is False         # t = 0 excluded
        assert oracle.hit_triangle([0, 0, 0], [1, 0, 0], tri, 0.0, fp64)[0] is False         # parallel
        assert oracle.hit_triangle([0, 0, 0], [0, 0, 0], tri, 0.0, fp64)[0] is False         # zero direction
        assert oracle.hit_triangle([0, 0, 0], [np.nan, 0, 1], tri, 0.0, fp64)[0] is False    # NaN direction
        # every dominant axis and both signs
        for axis in range(3):
            for sgn in (+1, -1):
                perm = np.roll(np.arange(3), axis + 1)
                t2 = tri[:, perm] * sgn
                d = np.zeros(3); d[perm.tolist().index(2)] = sgn
                o = np.zeros(3)
                o[perm.tolist().index(0)] = 0.25 * sgn
                assert oracle.hit_triangle(o, d, t2, 0.0, fp64) == (True, 5.0)


def test_hit_triangle_watertight_on_shared_edges_and_vertices():
    # Rays aimed exactly at shared edges / vertices of a fan of triangles must hit at least one.
    rng = np.random.default_rng(5)
    centre = np.float32([3.0, -2.0, 40.0])
    ring = [centre + np.float32([np.cos(a) * 7, np.sin(a) * 7, np.sin(3 * a)]) for a in
            np.linspace(0, 2 * np.pi, 9)[:-1]]
    tris = [np.stack([centre, ring[i], ring[(i + 1) % 8]]) for i in range(8)]
    o = np.float32([0.5, 0.25, -3.0])
    for k in range(400):
        i = k % 8
        s = np.float32(rng.random()) if k >= 8 else np.float32(0.0)       # s = 0: the shared vertex itself
        target = centre + s * (ring[i] - centre)                          # a point on the shared edge
        d = (target - o).astype(np.float32)                               # not normalised on purpose
        hits = [oracle.hit_triangle(o, d, t, 0.0, False)[0] for t in tris]
        assert any(hits)


# ------------------------------------------------------------- independent brute force (tiny)
def _reference_trace(scene, o, d, lam, seed):
    """Plain NumPy fp64 restatement of the state machine with Moeller-Trumbore and np.interp.
    Uses oracle.uniform (pinned by the KAT above) for the shared random stream."""
    tri, surf = scene.flat_triangles()
    tri = tri.astype(np.float64)
    grid = np.linspace(scene.lambda_min, scene.lambda_max, scene.n_lambda)
    out = []
    for i in range(len(lam)):
        oo, dd, b, last = o[i].astype(np.float64), d[i].astype(np.float64), 0, -1
        while True:
            best = (np.inf, -1)
            for k in range(len(tri)):
                if k == last:
                    continue
                h = _moller_trumbore(oo, dd, tri[k])
                if h is not None and h[0] > (0.0 if b == 0 else scene.t_min) and h[0] < best[0]:
                    best = (h[0], k)
            if best[1] < 0:
                out.append((6, -1, -1, b, oo)); break
            p = oo + best[0] * dd
            s = int(surf[best[1]])
            mat = scene.materials[scene.meshes[s]["material"]]
            eff = np.interp(float(lam[i]), grid, mat["table"].astype(np.float64))
            if mat["kind"] == MAT_ABSORBER:
                out.append((2, s, -1, b, p)); break
            if mat["kind"] == MAT_MIRROR:
                if not oracle.uniform(seed, i, b) < eff:
                    out.append((3, s, -1, b, p)); break
                t = tri[best[1]]
                n = np.cross(t[1] - t[0], t[2] - t[0]); n /= np.linalg.norm(n)
                dd = dd - 2 * (dd @ n) * n
                oo, last, b = p, best[1], b + 1
                if b == scene.max_bounces:
                    out.append((5, s, -1, b, p)); break
                continue
            f = scene.frames[scene.meshes[s]["frame"]]
            q = p - f["A"].astype(np.float64)
            iu = int(np.floor(q @ f["u"].astype(np.float64) / f["pitch_u"]))
            iv = int(np.floor(q @ f["v"].astype(np.float64) / f["pitch_v"]))
            if not (0 <= iu < f["nu"] and 0 <= iv < f["nv"]):
                out.append((4, s, -1, b, p)); break
            pix = f["pixel_base"] + iv * f["nu"] + iu
            out.append((0 if oracle.uniform(seed, i, b) < eff else 1, s, pix, b, p)); break
    return out


def _small_scene(cells=6):
    sc = wl.toy_rich_scene(tables="c2", cells=cells)
    return sc


@pytest.mark.parametrize("fp64", [True, False])
def test_state_machine_against_independent_brute_force(fp64):
    sc = _small_scene()
    src = TrackSource(600000, seed=3)                          # ~20 tracks; every 1000th photon
    o, d, lam = src.photons(np.arange(0, 600000, 1000))
    ref = _reference_trace(sc, o, d, lam, seed=11)
    got = oracle.trace_mesh(sc, o, d, lam, seed=11, fp64=fp64, n_threads=2)
    states = np.array([r[0] for r in ref])
    assert len(set(states)) >= 5                              # the sample exercises most terminal states
    n_bad = 0
    for i, r in enumerate(ref):
        same = (got.state[i], got.surface[i], got.pixel[i], got.bounces[i]) == r[:4]
        n_bad += not same
        if same:
            assert np.linalg.norm(got.pos[i] - r[4]) < (1e-8 if fp64 else 2e-3)
    assert n_bad <= (0 if fp64 else 1)                        # fp32 may flip one edge/pixel-boundary case


# --------------------------------------------------------------------------- P9 flat mirror
def test_p9_flat_mirror_is_textbook_image():
    z0 = 500.0
    sc = Scene()
    m_mir = sc.add_material(MAT_MIRROR, np.ones(N_LAMBDA))
    m_det = sc.add_material(MAT_DETECTOR, np.ones(N_LAMBDA))
    sc.add_mesh("mirror", [[-400, -400, z0], [400, -400, z0], [400, 400, z0], [-400, 400, z0]],
                [[0, 1, 2], [0, 2, 3]], m_mir)
    fr = sc.add_frame([-1000, -1000, -100.0], [1, 0, 0], [0, 1, 0], 4.0, 4.0, 500, 500, 0)
    sc.add_mesh("det", [[-1000, -1000, -100.0], [1000, -1000, -100.0], [1000, 1000, -100.0], [-1000, 1000, -100.0]],
                [[0, 1, 2], [0, 2, 3]], m_det, frame=fr)
    rng = np.random.default_rng(6)
    n = 500
    d = np.stack([rng.uniform(-0.5, 0.5, n), rng.uniform(-0.5, 0.5, n), np.ones(n)], axis=1)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    o = np.zeros((n, 3))
    lam = np.full(n, 400.0)
    for fp64 in (True, False):
        r = oracle.trace_mesh(sc, o, d, lam, seed=0, fp64=fp64)
        assert np.all(r.state == oracle.DETECTED) and np.all(r.bounces == 1)
        # straight ray from the image source (0,0,2 z0) with direction (dx,dy,-dz) to z = -100
        d32 = d.astype(np.float32).astype(np.float64)
        t = (2 * z0 + 100.0) / d32[:, 2]
        want = np.stack([t * d32[:, 0], t * d32[:, 1], np.full(n, -100.0)], axis=1)
        assert np.abs(r.pos - want).max() < (1e-9 if fp64 else 5e-4)
        np.testing.assert_allclose(r.dir, d32 * [1, 1, -1], atol=1e-12 if fp64 else 2e-7)
        assert np.array_equal(r.pixel, (np.floor((want[:, 1] + 1000) / 4) * 500 + np.floor((want[:, 0] + 1000) / 4)).astype(np.int32)) \
            or not fp64


# ------------------------------------------------------------- P3 / P5 / P6 / P8 the toy RICH
@pytest.fixture(scope="module")
def c1():
    w = wl.make_config("C1", n=20000)
    o, d, lam = w.photon_range(0, w.n)
    return w, o, d, lam


def test_p1_generator_cherenkov_angle(c1):
    _, o, d, lam = c1
    th = cherenkov_angle()
    g = _golden(os.path.join(os.path.dirname(__file__), "golden", "c1_focal_ring.txt"))
    assert abs(th - g["theta_c_rad"][0]) < g["theta_c_rad"][1]
    assert abs(np.tan(th) - g["tan_theta_c"][0]) < g["tan_theta_c"][1]
    assert abs(np.cos(th) - 1 / 1.0014) < 1e-15               # cos(theta_c) = 1/(n beta)
    ang = np.arccos(np.clip(d.astype(np.float64) @ [0, 0, 1.0], -1, 1))
    assert np.abs(ang - th).max() < 2e-6                      # fp32 rounding of the direction
    phi = np.arctan2(d[:, 1], d[:, 0])
    assert abs(np.mean(np.cos(phi))) < 0.03 and abs(np.mean(np.sin(phi))) < 0.03   # azimuth uniform
    assert np.all(o == 0) and lam.min() >= 200 and lam.max() <= 600
    assert abs(lam.mean() - 400) < 4 * 400 / np.sqrt(12 * len(lam))
    # track generator: angle to the *track* is theta_c(beta) for every photon
    src = TrackSource(5000, seed=1, beta_lo=0.9999)
    ids = np.arange(5000)
    o2, d2, _ = src.photons(ids)
    gstep = np.searchsorted(src.offsets, ids, side="right") - 1
    _, w, beta = src.tracks(gstep // src.n_steps)
    ang = np.arccos(np.clip(np.sum(d2.astype(np.float64) * w, axis=1), -1, 1))
    assert np.abs(ang - cherenkov_angle(beta=beta)).max() < 3e-6


def test_p13_generator_distributions():
    src = TrackSource(2000000, seed=2)
    counts = np.diff(src.offsets)                              # ~69k steps: 4 sigma on mean / variance
    assert abs(counts.mean() - 30) < 0.09 and abs(counts.var() - 30) < 0.7     # Poisson(30)
    _, _, lam = src.photons(np.arange(0, 200000, 4))
    # density ~ 1/lambda^2 on [200,600]: E[lambda] = 300 ln 3, E[1/lambda] = (1/200^2-1/600^2)/2 * 300
    assert abs(lam.astype(np.float64).mean() - 300 * np.log(3)) < 1.5
    assert abs((1 / lam.astype(np.float64)).mean() - 300 * 0.5 * (1 / 200 ** 2 - 1 / 600 ** 2)) < 2e-5
    o, w, _ = src.tracks(np.arange(2000))
    assert np.all(np.hypot(o[:, 0], o[:, 1]) <= 100) and np.all(o[:, 2] == 0)
    assert np.all(np.arccos(w[:, 2]) <= 0.250 + 1e-12)
    # any id subset reproduces the same photons (ids are the only key)
    a = src.photons(np.arange(1000, 2000))
    b = src.photons(np.arange(1000, 2000)[::-1])
    for x, y in zip(a, b):
        assert np.array_equal(x, y[::-1])


def test_p3_focal_ring_analytic(c1, golden_dir):
    w, o, d, lam = c1
    g = _golden(os.path.join(golden_dir, "c1_focal_ring.txt"))
    r = oracle.trace_analytic_toy(w.scene, o, d, lam, seed=0)
    info = w.scene.info
    closed = 0.5 * info["R"] * np.tan(cherenkov_angle())
    assert abs(closed - g["closed_form_radius_mm"][0]) < g["closed_form_radius_mm"][1]
    on_det = r.state <= oracle.QE_REJECTED
    assert on_det.sum() > 0.85 * w.n
    q = r.pos[on_det] - info["D"]
    a, b = q @ info["du"], q @ info["dv"]
    assert np.abs(q @ np.cross(info["du"], info["dv"])).max() < 1e-9       # hits lie in the detector plane
    rad = np.hypot(a, b)
    assert abs(rad.mean() / closed - 1) < 3e-3                             # ring of radius ~ (R/2) tan(theta_c)
    chk = dict(mean_radius_mm=rad.mean(), radius_min_mm=rad.min(), radius_max_mm=rad.max(),
               u_semi_axis_mm=np.abs(a).max(), v_min_mm=b.min(), v_max_mm=b.max())
    for k, v in chk.items():
        assert abs(v - g[k][0]) <= g[k][1], (k, v)
    pix = r.pixel[on_det]
    assert len(np.unique(pix)) == int(g["distinct_pixels"][0])
    assert (pix % 208).min() == g["iu_min"][0] and (pix % 208).max() == g["iu_max"][0]
    assert (pix // 208).min() == g["iv_min"][0] and (pix // 208).max() == g["iv_max"][0]
    # path lengths ~ 1200.9 mm to the mirror and ~ 1199.1 mm on to the detector
    assert np.all(r.bounces[on_det] == 1)


def test_p5_tessellated_vs_analytic_sphere(c1, golden_dir):
    w, o, d, lam = c1
    g = _golden(os.path.join(golden_dir, "c1_focal_ring.txt"))
    ana = oracle.trace_analytic_toy(w.scene, o, d, lam, seed=0)
    for fp64 in (True, False):
        mesh = oracle.trace_mesh(w.scene, o, d, lam, seed=0, fp64=fp64)
        assert np.array_equal(mesh.state, ana.state)           # same Philox stream, same tables
        on_det = ana.state <= oracle.QE_REJECTED
        dev = np.linalg.norm(mesh.pos[on_det] - ana.pos[on_det], axis=1)
        rc = w.scene.info["facet_circumradius"]
        assert abs(rc - g["tess_max_dev_mm"][0]) < 1e-3
        assert dev.max() <= rc and 2.5 < np.sqrt((dev ** 2).mean()) < 4.0
        ddev = np.arccos(np.clip(np.sum(mesh.dir[on_det] * ana.dir[on_det], axis=1), -1, 1))
        assert ddev.max() <= 2 * rc / w.scene.info["R"] * 1.01
        # photons absorbed on the mirror stop at the mirror hit: sag error <= rc^2 / (2R)
        on_mir = ana.state == oracle.ABSORBED_MIRROR
        mdev = np.linalg.norm(mesh.pos[on_mir] - ana.pos[on_mir], axis=1)
        assert mdev.max() <= g["tess_mirror_dev_mm"][0] * 1.02
        # detected pixels differ, but the ring radius agrees to the facet blur
        q = mesh.pos[on_det] - w.scene.info["D"]
        assert abs(np.hypot(q @ w.scene.info["du"], q @ w.scene.info["dv"]).mean() - 63.70) < 0.1


def test_p6_binomial_counts(c1):
    w, _, _, _ = c1
    n = 100000
    o, d, lam = w.photon_range(0, n)
    r = oracle.trace_analytic_toy(w.scene, o, d, lam, seed=0)
    cnt = np.bincount(r.state, minlength=7)
    assert cnt.sum() == n
    # reflectivity 0.9 flat, QE 0.25 flat: detected 22 500 +- 132, QE-rejected 67 500, mirror-absorbed 10 000
    assert abs(cnt[oracle.DETECTED] - 0.9 * 0.25 * n) < 4 * np.sqrt(n * 0.225 * 0.775)
    assert abs(cnt[oracle.QE_REJECTED] - 0.9 * 0.75 * n) < 4 * np.sqrt(n * 0.675 * 0.325)
    assert abs(cnt[oracle.ABSORBED_MIRROR] - 0.1 * n) < 4 * np.sqrt(n * 0.1 * 0.9)
    assert cnt[oracle.ESCAPED] == 0 and cnt[oracle.DETECTOR_DEAD] == 0 and cnt[oracle.ABSORBED_SURFACE] == 0
    # a different seed gives a different but statistically equal split
    r2 = oracle.trace_analytic_toy(w.scene, o, d, lam, seed=1)
    assert not np.array_equal(r.state, r2.state)
    assert abs(int(np.sum(r2.state == 0)) - 0.225 * n) < 4 * np.sqrt(n * 0.225 * 0.775)


def test_p8_retro_reflection_from_centre_of_curvature():
    sc = wl.toy_rich_scene(tables="flat")
    sc.materials[1]["table"][:] = 1.0                          # perfect mirror for this pin
    g = sc.info
    rng = np.random.default_rng(8)
    n = 300
    tgt = g["V"] + rng.uniform(-350, 350, (n, 1)) * g["ex"] + rng.uniform(-350, 350, (n, 1)) * g["ey"]
    d = tgt - g["C"]
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    o = np.tile(g["C"], (n, 1))
    lam = np.full(n, 400.0)
    # the detector and the enclosure stand between C and the mirror: trace the mirror alone
    o32, d32 = o.astype(np.float32).astype(np.float64), d.astype(np.float32).astype(np.float64)
    only = Scene()
    mm = only.add_material(MAT_MIRROR, np.ones(N_LAMBDA))
    only.add_mesh("mirror", sc.meshes[0]["vertices"], sc.meshes[0]["indices"], mm)
    only.max_bounces = 1
    r = oracle.trace_mesh(only, o, d, lam, fp64=True)
    ok = r.state == oracle.BOUNCE_LIMIT
    assert ok.sum() > 0.8 * n
    t_hit = np.linalg.norm(r.pos[ok] - o32[ok], axis=1)
    rc = g["facet_circumradius"]
    assert np.abs(t_hit - g["R"]).max() < rc ** 2 / (2 * g["R"]) * 1.05     # chord sag
    # distance from C to the reflected line
    back = np.linalg.norm(np.cross(o32[ok] - r.pos[ok], r.dir[ok]), axis=1) / np.linalg.norm(r.dir[ok], axis=1)
    assert back.max() < 2 * rc
    # analytic sphere: t = R exactly and the ray returns through C
    only_ana_pos = o32 + g["R"] * d32
    first = oracle.trace_analytic_toy(_mirror_only_toy(sc), o, d, lam, seed=0, with_box=False, det_half=-1.0)
    ok2 = first.state == oracle.BOUNCE_LIMIT
    assert np.abs(first.pos[ok2] - only_ana_pos[ok2]).max() < 1e-3          # fp32 C is 6e-5 off the true centre
    back2 = np.linalg.norm(np.cross(o32[ok2] - first.pos[ok2], first.dir[ok2]), axis=1)
    assert back2.max() < 1e-3


def _mirror_only_toy(sc):
    import copy
    c = copy.copy(sc)
    c.max_bounces = 1
    return c


# ---------------------------------------------------------------- P4 conservation, P12 invariance
def test_p4_conservation_and_hitmap(c1):
    w = wl.make_config("C3", n=600000)                         # ~20 tracks
    ids = np.arange(0, w.n, 200, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    r = oracle.trace_mesh(w.scene, o, d, lam, seed=5, ids=ids)
    assert int(r.counters[:7].sum()) == len(ids)
    assert np.array_equal(r.counters[:7], np.bincount(r.state, minlength=7))
    det = r.state == oracle.DETECTED
    assert int(r.hitmap.sum()) == int(det.sum()) == int(r.counters[0])
    assert np.array_equal(r.hitmap, np.bincount(r.pixel[det], minlength=w.scene.n_pixels))
    assert int(r.counters[7]) == int(r.segments.sum())
    assert np.all(r.pixel[r.state > oracle.QE_REJECTED] == -1) and np.all(r.pixel[r.state <= 1] >= 0)
    assert np.all(r.surface[r.state == oracle.ESCAPED] == -1)
    # C3 exercises several terminal states (tracks up to 250 mrad miss the mirror or the detector)
    assert len(np.unique(r.state)) >= 4


def test_p12_order_invariance_and_fp32_adequacy():
    w = wl.make_config("C3", n=600000)
    ids = np.arange(0, w.n, 150, dtype=np.uint64)
    n = len(ids)
    o, d, lam = w.photons(ids)
    base = oracle.trace_mesh(w.scene, o, d, lam, seed=9, ids=ids)
    # photon order permuted, ids carried: identical per-id results
    perm = np.random.default_rng(0).permutation(n)
    p = oracle.trace_mesh(w.scene, o[perm], d[perm], lam[perm], seed=9, ids=ids[perm])
    assert len(np.unique(base.state)) >= 5
    for k in ("state", "pixel", "surface", "bounces", "tri", "pos", "dir"):
        assert np.array_equal(p[k], base[k][perm]), k
    assert np.array_equal(p.hitmap, base.hitmap)
    # chunking with id_base: identical (contiguous ids 1000..1999 traced as 2 chunks vs explicit ids)
    cid = np.arange(1000, 2000, dtype=np.uint64)
    co, cd, cl = w.photons(cid)
    whole = oracle.trace_mesh(w.scene, co, cd, cl, seed=9, ids=cid)
    c0 = oracle.trace_mesh(w.scene, co[:300], cd[:300], cl[:300], seed=9, id_base=1000)
    c1_ = oracle.trace_mesh(w.scene, co[300:], cd[300:], cl[300:], seed=9, id_base=1300)
    assert np.array_equal(np.concatenate([c0.state, c1_.state]), whole.state)
    assert np.array_equal(c0.hitmap + c1_.hitmap, whole.hitmap)
    shifted = oracle.trace_mesh(w.scene, co, cd, cl, seed=9, id_base=0)     # other ids: other draws
    assert not np.array_equal(shifted.state, whole.state)
    # thread count does not matter
    one = oracle.trace_mesh(w.scene, o[:500], d[:500], lam[:500], seed=9, ids=ids[:500], n_threads=1)
    assert np.array_equal(one.state, base.state[:500]) and np.array_equal(one.pos, base.pos[:500])
    # fp32 contract vs fp64: same facet except on ~1e-6 of photons, positions within 1e-3 mm
    f64 = oracle.trace_mesh(w.scene, o, d, lam, seed=9, ids=ids, fp64=True)
    same = (f64.tri == base.tri) & (f64.state == base.state)
    assert (~same).sum() <= 2
    assert np.abs(f64.pos[same] - base.pos[same]).max() < 1e-3
    ang = np.linalg.norm(f64.dir[same] - base.dir[same], axis=1)
    assert ang.max() < 1e-6


# ------------------------------------------------------------------------------- edge cases
def test_edge_cases():
    sc = _small_scene()
    z = np.zeros((0, 3), np.float32)
    r = oracle.trace_mesh(sc, z, z, np.zeros(0, np.float32))
    assert len(r.state) == 0 and r.hitmap.sum() == 0 and r.counters.sum() == 0
    # NaN / zero directions end ESCAPED at the origin; a photon leaving through no surface too
    nob = wl.toy_rich_scene(cells=4, enclosure=False)
    o = np.zeros((4, 3), np.float32)
    d = np.float32([[np.nan, 0, 1], [0, 0, 0], [0, 0, -1], [0, 0, 1]])
    r = oracle.trace_mesh(nob, o, d, np.full(4, 400.0), seed=0)
    assert list(r.state[:3]) == [oracle.ESCAPED] * 3 and np.all(r.surface[:3] == -1)
    assert np.all(r.pos[:3] == 0) and r.state[3] != oracle.ESCAPED
    assert r.segments[3] >= 1 and r.bounces[0] == 0
    # with the enclosure the backward photon is absorbed on the box
    r2 = oracle.trace_mesh(sc, o[2:3], d[2:3], [400.0])
    assert r2.state[0] == oracle.ABSORBED_SURFACE and sc.meshes[r2.surface[0]]["name"] == "enclosure"


def test_bounce_limit_between_parallel_mirrors():
    sc = Scene()
    m = sc.add_material(MAT_MIRROR, np.ones(N_LAMBDA))
    for z in (-10.0, 10.0):
        sc.add_mesh("m", [[-50, -50, z], [50, -50, z], [50, 50, z], [-50, 50, z]], [[0, 1, 2], [0, 2, 3]], m)
    for fp64 in (True, False):
        r = oracle.trace_mesh(sc, [[0, 0, 0]], [[0.01, 0.0, 1.0]], [300.0], fp64=fp64)
        assert r.state[0] == oracle.BOUNCE_LIMIT and r.bounces[0] == 16 and r.segments[0] == 16
        # 16 reflections: 10 mm up, then 15 x 20 mm; x advances by 0.01 per unit z
        assert abs(r.pos[0][0] - 0.01 * (10 + 15 * 20)) < 1e-4 and abs(abs(r.pos[0][2]) - 10) < 1e-6
        assert r.dir[0][2] * r.pos[0][2] < 0                   # direction already reflected back inwards
    # reflectivity 0 never reflects; reflectivity 1 always does (strict u < value)
    sc.materials[0]["table"][:] = 0.0
    r = oracle.trace_mesh(sc, [[0, 0, 0]], [[0.0, 0.0, 1.0]], [300.0])
    assert r.state[0] == oracle.ABSORBED_MIRROR and r.bounces[0] == 0
