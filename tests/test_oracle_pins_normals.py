"""Pins of the oracle's SURVEY.md 8(f) row f3 (interpolated vertex normals) against things other than
the oracle: NumPy fp64 barycentric interpolation from a Moller-Trumbore hit, the law of reflection, and the closed
form that makes the row worth having -- on a tessellated sphere whose vertex normals point at the centre of
curvature the interpolated normal at a facet point p is exactly (C - p)/|C - p|, so the mesh reproduces the analytic
sphere's reflected directions and focal ring instead of blurring them by the facet size.
CPU only.  P-numbers continue DESIGN.md section 6."""
import numpy as np
import pytest

import oracle
import workloads as wl
from workloads.scenes import MAT_MIRROR, N_LAMBDA, Scene, toy_rich_scene


def _unit(v):
    v = np.asarray(v, np.float64)
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _random_triangle(rng):
    # roughly face-on to rays from near the origin: fp32 edge functions cancel badly on a triangle seen edge-on,
    # which is a property of the test of DESIGN.md 3.3, not of the interpolation pinned here
    tri = rng.uniform(-5, 5, (3, 3)) * np.array([1, 1, 0.2]) + np.array([0, 0, 20.0])
    vn = _unit(rng.normal(size=(3, 3)) * 0.2 + np.array([0, 0, -1.0]))
    return tri.astype(np.float32), vn.astype(np.float32)


# ------------------------------------------------------------------ P19 the interpolation itself
@pytest.mark.parametrize("fp64", [False, True])
def test_p19_weights_belong_to_their_vertices(fp64):
    """A ray aimed at wa*a + wb*b + wc*c: the edge functions are proportional to (wa, wb, wc) in that order, and
    the normal is the normalised weighted sum of (na, nb, nc) computed in NumPy fp64."""
    rng = np.random.default_rng(19)
    tol = 1e-12 if fp64 else 2e-5
    for _ in range(300):
        tri, vn = _random_triangle(rng)
        w = rng.dirichlet([1, 1, 1])
        target = w @ tri.astype(np.float64)
        o = rng.uniform(-3, 3, 3).astype(np.float32)
        d = _unit(target - o).astype(np.float32)
        n, uvw = oracle.shading_normal(o, d, tri, vn, fp64=fp64)
        # the float32 direction misses `target` slightly: recompute the true barycentrics of the actual ray in fp64
        a, b, c = tri.astype(np.float64)
        M = np.stack([b - a, c - a, -d.astype(np.float64)], axis=1)
        s, t, _ = np.linalg.solve(M, o.astype(np.float64) - a)
        want_w = np.array([1 - s - t, s, t])
        a2 = 0.5 * np.linalg.norm(np.cross(b - a, c - a))
        if a2 < 2.0:
            continue                                            # slivers: same cancellation
        assert np.allclose(uvw / uvw.sum(), want_w, atol=tol * 10)
        want = _unit(want_w @ vn.astype(np.float64))
        assert np.allclose(n, want, atol=tol * 10) or np.allclose(n, -want, atol=tol * 10)
        assert abs(np.linalg.norm(n) - 1) < (1e-12 if fp64 else 3e-7)


def test_p19_special_cases():
    rng = np.random.default_rng(20)
    tri, vn = _random_triangle(rng)
    a, b, c = tri.astype(np.float64)
    o = np.zeros(3, np.float32)
    # equal vertex normals: the weights drop out
    same = np.tile(_unit([0.1, -0.2, -1.0]), (3, 1)).astype(np.float32)
    n, _ = oracle.shading_normal(o, _unit((a + b + c) / 3 + [0.3, 0.1, 0]).astype(np.float32), tri, same)
    assert np.allclose(n, same[0], atol=3e-7) or np.allclose(n, -same[0], atol=3e-7)
    # centroid: the normalised mean; near a vertex: that vertex's normal; on an edge: only its two ends count
    n, _ = oracle.shading_normal(o, _unit((a + b + c) / 3).astype(np.float32), tri, vn, fp64=True)
    assert np.allclose(np.abs(n), np.abs(_unit(vn.astype(np.float64).sum(axis=0))), atol=1e-6)
    for k, v in enumerate((a, b, c)):
        inside = v + 1e-4 * ((a + b + c) / 3 - v)
        n, _ = oracle.shading_normal(o, _unit(inside).astype(np.float32), tri, vn, fp64=True)
        assert np.allclose(np.abs(n), np.abs(vn[k].astype(np.float64)), atol=1e-3)
    n, uvw = oracle.shading_normal(o, _unit(0.5 * (a + b) + 1e-6 * (c - a)).astype(np.float32), tri, vn, fp64=True)
    assert abs(uvw[2] / uvw.sum()) < 1e-4
    assert np.allclose(np.abs(n), np.abs(_unit(vn[0].astype(np.float64) * uvw[0] + vn[1] * uvw[1])), atol=1e-4)
    # no vertex normals (all zero): the face normal; from the back: the same normal up to sign
    d = _unit((a + b + c) / 3).astype(np.float32)
    n0, _ = oracle.shading_normal(o, d, tri, np.zeros((3, 3), np.float32))
    assert np.allclose(np.abs(n0), np.abs(oracle.face_normal(tri)), atol=1e-7)
    far = (2.5 * (a + b + c) / 3).astype(np.float32)
    nf, _ = oracle.shading_normal(o, d, tri, vn)
    nb, _ = oracle.shading_normal(far, -d, tri, vn)
    assert np.allclose(np.abs(nf), np.abs(nb), atol=2e-5)
    assert oracle.shading_normal(o, np.float32([0, 0, -1]), tri, vn) is None          # a miss


# ------------------------------------------- P20 independent NumPy brute force with vertex normals
def test_p20_mirror_patch_against_numpy():
    """One mirror of R = 1 made of a 6x6 wavy patch with random vertex normals: the photon's record after the first
    reflection (it then escapes: position = the hit, direction = the reflected one, R17) against
    Moller-Trumbore + barycentric interpolation + d - 2(d.n)n in NumPy fp64."""
    rng = np.random.default_rng(21)
    k = 6
    xs = np.linspace(-30, 30, k + 1)
    X, Y = np.meshgrid(xs, xs)
    verts = np.stack([X.ravel(), Y.ravel(), 100 + 2 * np.sin(X.ravel() / 9) + rng.uniform(-0.5, 0.5, X.size)], axis=1)
    idx = []
    for j in range(k):
        for i in range(k):
            v00 = j * (k + 1) + i
            idx += [[v00, v00 + k + 2, v00 + 1], [v00, v00 + k + 1, v00 + k + 2]]
    vn = _unit(rng.normal(size=verts.shape) * 0.15 + np.array([0, 0, -1.0]))
    sc = Scene()
    m = sc.add_material(MAT_MIRROR, np.ones(N_LAMBDA))
    sc.add_mesh("patch", verts, idx, m, vertex_normals=vn)
    n = 3000
    d = _unit(np.stack([rng.uniform(-0.25, 0.25, n), rng.uniform(-0.25, 0.25, n), np.ones(n)], axis=1)).astype(np.float32)
    o = rng.uniform(-2, 2, (n, 3)).astype(np.float32)
    lam = np.full(n, 400.0, np.float32)
    mesh = sc.meshes[0]
    tri = mesh["vertices"][mesh["indices"].astype(np.int64)].astype(np.float64)       # (T,3,3)
    tvn = mesh["vertex_normals"][mesh["indices"].astype(np.int64)].astype(np.float64)
    got = oracle.trace_mesh(sc, o, d, lam, seed=1, fp64=True)
    got32 = oracle.trace_mesh(sc, o, d, lam, seed=1)
    hit = 0
    for i in range(n):
        oo, dd = o[i].astype(np.float64), d[i].astype(np.float64)
        a, e1, e2 = tri[:, 0], tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0]
        p = np.cross(dd, e2)
        det = np.einsum("ij,ij->i", e1, p)
        tv = oo - a
        u = np.einsum("ij,ij->i", tv, p) / det
        q = np.cross(tv, e1)
        v = np.einsum("ij,j->i", q, dd) / det
        t = np.einsum("ij,ij->i", e2, q) / det
        ok = (u >= 0) & (v >= 0) & (u + v <= 1) & (t > 0)
        if not ok.any():
            assert got.state[i] == oracle.ESCAPED and got.bounces[i] == 0
            continue
        kbest = np.flatnonzero(ok)[np.argmin(t[ok])]
        margin = min(u[kbest], v[kbest], 1 - u[kbest] - v[kbest])
        if margin < 1e-6:
            continue                                            # on an edge: either neighbour is a valid answer
        hit += 1
        nn = _unit((1 - u[kbest] - v[kbest]) * tvn[kbest, 0] + u[kbest] * tvn[kbest, 1] + v[kbest] * tvn[kbest, 2])
        r = dd - 2 * (dd @ nn) * nn
        assert got.tri[i] == kbest
        if got.bounces[i] == 1:                                 # the reflected ray left the patch
            assert np.allclose(got.dir[i], r, atol=1e-9) and got.state[i] == oracle.ESCAPED
            assert np.allclose(got.pos[i], oo + t[kbest] * dd, atol=1e-7)
            if got32.bounces[i] == 1 and got32.tri[i] == kbest:
                assert np.allclose(got32.dir[i], r, atol=2e-5)
    assert hit > 2000 and (got.bounces == 1).sum() > 1500


# ------------------------------ P21 the closed form: sphere mesh + exact vertex normals == sphere
@pytest.fixture(scope="module")
def c1_smooth():
    w = wl.make_config("C1", n=20000)
    o, d, lam = w.photon_range(0, w.n)
    sc = toy_rich_scene("flat", smooth=True)
    return w, sc, o, d, lam


def test_p21_smooth_sphere_mesh_reproduces_the_analytic_sphere(c1_smooth):
    w, sc, o, d, lam = c1_smooth
    ana = oracle.trace_analytic_toy(w.scene, o, d, lam, seed=0)
    flat = oracle.trace_mesh(w.scene, o, d, lam, seed=0)
    R, rc = sc.info["R"], sc.info["facet_circumradius"]
    # interpolated normal at facet point p = (C - p)/|C - p| exactly; p lies s <= rc^2/2R in front of the sphere, so the
    # normal is off by s sin(incidence)/R and the reflected direction by twice that: (rc/R)^2 sin(0.35) = 1.9e-6 rad
    bound = (rc / R) ** 2 * np.sin(0.35)
    for fp64, dir_tol in ((True, bound), (False, bound + 1e-6)):
        sm = oracle.trace_mesh(sc, o, d, lam, seed=0, fp64=fp64)
        assert np.array_equal(sm.state, ana.state)
        on_det = ana.state <= oracle.QE_REJECTED
        ddev = np.linalg.norm(np.cross(sm.dir[on_det], ana.dir[on_det]), axis=1)     # sin(angle): arccos is blind below 1e-4
        assert 0.2 * bound < ddev.max() < dir_tol, ddev.max()
        dev = np.linalg.norm(sm.pos[on_det] - ana.pos[on_det], axis=1)
        assert dev.max() < 0.02, dev.max()                      # vs the facet circumradius 5.657 mm with face normals
    fdev = np.linalg.norm(flat.pos[on_det] - ana.pos[on_det], axis=1)
    assert fdev.max() > 100 * dev.max() and fdev.max() <= rc
    # the ring: same pixels as the analytic sphere for all but photons within 0.02 mm of a pixel boundary
    assert np.mean(sm.pixel[on_det] != ana.pixel[on_det]) < 0.02
    assert np.mean(flat.pixel[on_det] != ana.pixel[on_det]) > 0.5
    q = sm.pos[on_det] - sc.info["D"]
    rad = np.hypot(q @ sc.info["du"], q @ sc.info["dv"])
    qa = ana.pos[on_det] - sc.info["D"]
    assert abs(rad.mean() - np.hypot(qa @ sc.info["du"], qa @ sc.info["dv"]).mean()) < 1e-3


def test_p21_meshes_without_vertex_normals_are_unchanged(c1_smooth):
    """The detector and the enclosure of the smooth scene carry no vertex normals, and a scene with none at all takes
    the face-normal path: same records as before the row existed (zero vertex normals == face normal)."""
    w, sc, o, d, lam = c1_smooth
    base = oracle.trace_mesh(w.scene, o[:3000], d[:3000], lam[:3000], seed=0)
    tri, _ = w.scene.flat_triangles()
    zeros = oracle.trace_mesh_arrays(*_arrays(w.scene), o[:3000], d[:3000], lam[:3000], seed=0,
                                     tri_vnormal=np.zeros((len(tri), 9), np.float32))
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir", "tri"):
        assert np.array_equal(base[k], zeros[k]), k


def _arrays(scene):
    tri, tri_surface = scene.flat_triangles()
    frames = (oracle.Frame * max(1, len(scene.frames)))(*[oracle.make_frame(f) for f in scene.frames])
    return (np.ascontiguousarray(tri.reshape(-1, 9)), tri_surface,
            np.ascontiguousarray([m["material"] for m in scene.meshes], dtype=np.uint32),
            np.ascontiguousarray([m["frame"] for m in scene.meshes], dtype=np.int32),
            np.ascontiguousarray([m["kind"] for m in scene.materials], dtype=np.uint32),
            np.ascontiguousarray(np.stack([m["table"] for m in scene.materials]), dtype=np.float32),
            scene.lambda_min, scene.lambda_max, frames, len(scene.frames), scene.max_bounces, scene.t_min, scene.n_pixels)
