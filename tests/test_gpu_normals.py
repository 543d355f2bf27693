"""GPU parity for SURVEY.md 8(f) row f3: interpolated vertex normals through the C ABI against the
oracle on the same seeded inputs.  Both sides evaluate the same fp32 sequence (edge functions of the winning triangle,
weighted sum, IEEE sqrt and divide), so the bar is the one of tests/test_gpu_parity.py and the expectation is zero
mismatches with bit-identical positions and directions."""
import ctypes as C

import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl
from paper_2309_12496_b200 import opx
from workloads.scenes import MAT_ABSORBER, MAT_DETECTOR, MAT_MIRROR, N_LAMBDA, Scene, toy_rich_scene

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def _host(out):
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def _unit(v):
    v = np.asarray(v, np.float64)
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _assert_identical(got, ref, n):
    for k in ("state", "surface", "pixel", "bounces"):
        assert np.array_equal(got[k][:n], ref[k]), k
    assert np.array_equal(got["pos"][:n].astype(np.float64), ref["pos"])
    assert np.array_equal(got["dir"][:n].astype(np.float64), ref["dir"], equal_nan=True)
    assert np.array_equal(got["hitmap"], ref["hitmap"]) and np.array_equal(got["counters"].astype(np.uint64), ref["counters"])


@pytest.fixture(scope="module")
def smooth():
    sc = toy_rich_scene("c2", smooth=True)
    return sc, pkg.Scene(sc).build()


def test_smooth_toy_mirror_full_mesh_parity(smooth):
    """The C1/C2 scene (20 014 triangles) with vertex normals on the mirror: 2e4 C3-style photons, every output."""
    sc, gs = smooth
    w = wl.make_config("C3", n=4_000_000)
    ids = np.arange(0, w.n, 200, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=12))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=12)
    _assert_identical(got, ref, len(ids))
    assert len(np.unique(ref["state"])) >= 4 and (ref["bounces"] >= 1).mean() > 0.5


def test_smooth_mirror_sharpens_the_ring_on_the_gpu(smooth):
    """The closed form behind the row, on the GPU result itself: with vertex normals (C - v)/R the C1 ring lands in the
    analytic sphere's pixels (P21), which face normals miss by up to the 5.66 mm facet circumradius."""
    sc, gs = smooth
    w = wl.make_config("C1", n=20_000)
    o, d, lam = w.photon_range(0, w.n)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=0))
    ana = oracle.trace_analytic_toy(sc, o, d, lam, seed=0)
    assert np.array_equal(got["state"], ana.state)
    on_det = ana.state <= 1
    assert np.linalg.norm(got["pos"][on_det] - ana.pos[on_det], axis=1).max() < 0.02
    assert np.linalg.norm(np.cross(got["dir"][on_det].astype(np.float64), ana.dir[on_det]), axis=1).max() < 3e-6
    assert np.mean(got["pixel"][on_det] != ana.pixel[on_det]) < 0.02
    flat = pkg.Scene(toy_rich_scene("c2")).build()
    f = _host(flat.propagate(*_dev(o, d, lam), seed=0))
    assert np.mean(f["pixel"][on_det] != ana.pixel[on_det]) > 0.5


def _wavy_cavity(rng, k=24, with_normals=(True, True)):
    """Two facing wavy mirror patches (random vertex normals on one or both), a detector strip and an absorbing box:
    photons bounce between the mirrors up to the limit, leak to the detector or the box."""
    sc = Scene()
    m_abs = sc.add_material(MAT_ABSORBER, np.zeros(N_LAMBDA))
    m_mir = sc.add_material(MAT_MIRROR, np.linspace(0.95, 1.0, N_LAMBDA))
    m_det = sc.add_material(MAT_DETECTOR, np.linspace(0.3, 0.8, N_LAMBDA))
    xs = np.linspace(-60, 60, k + 1)
    X, Y = np.meshgrid(xs, xs)
    idx = []
    for j in range(k):
        for i in range(k):
            v00 = j * (k + 1) + i
            idx += [[v00, v00 + k + 2, v00 + 1], [v00, v00 + k + 1, v00 + k + 2]]
    for z0, sgn, has in ((40.0, -1.0, with_normals[0]), (-40.0, 1.0, with_normals[1])):
        verts = np.stack([X.ravel(), Y.ravel(), z0 + 1.5 * np.sin(X.ravel() / 11) * np.cos(Y.ravel() / 7) + rng.uniform(-0.3, 0.3, X.size)], axis=1)
        vn = _unit(rng.normal(size=verts.shape) * 0.05 + np.array([0, 0, sgn]))
        sc.add_mesh("mirror", verts, idx, m_mir, vertex_normals=vn if has else None)
    fr = sc.add_frame([70.0, -60, -40], [0, 1, 0], [0, 0, 1], 2.0, 2.0, 60, 40, 0)
    sc.add_mesh("det", [[70.0, -60, -40], [70.0, 60, -40], [70.0, 60, 40], [70.0, -60, 40]], [[0, 1, 2], [0, 2, 3]], m_det, frame=fr)
    lo, hi = np.array([-100.0, -100, -100]), np.array([100.0, 100, 100])
    c = np.array([[lo[0], lo[1], lo[2]], [hi[0], lo[1], lo[2]], [hi[0], hi[1], lo[2]], [lo[0], hi[1], lo[2]],
                  [lo[0], lo[1], hi[2]], [hi[0], lo[1], hi[2]], [hi[0], hi[1], hi[2]], [lo[0], hi[1], hi[2]]])
    box = [[0, 1, 2], [0, 2, 3], [4, 6, 5], [4, 7, 6], [0, 4, 5], [0, 5, 1], [1, 5, 6], [1, 6, 2], [2, 6, 7], [2, 7, 3], [3, 7, 4], [3, 4, 0]]
    sc.add_mesh("box", c, box, m_abs)
    return sc


@pytest.mark.parametrize("with_normals", [(True, True), (True, False)])
def test_multi_bounce_cavity_with_random_vertex_normals(with_normals):
    """Up to 16 reflections about interpolated normals (errors would compound), meshes with and without vertex
    normals in one scene, every terminal state; BVH == GPU all-triangle loop on ten times as many photons."""
    rng = np.random.default_rng(33)
    sc = _wavy_cavity(rng, with_normals=with_normals)
    gs = pkg.Scene(sc).build()
    n = 30_000
    d = _unit(np.stack([rng.uniform(-0.6, 0.6, n), rng.uniform(-0.4, 0.4, n), rng.choice([-1.0, 1.0], n)], axis=1)).astype(np.float32)
    o = rng.uniform(-20, 20, (n, 3)).astype(np.float32)
    lam = rng.uniform(200, 600, n).astype(np.float32)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=7))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=7)
    _assert_identical(got, ref, n)
    assert ref["bounces"].max() == 16 and (ref["state"] == 5).sum() > 10 and (ref["state"] == 0).sum() > 100
    assert len(np.unique(ref["state"])) >= 5
    n2 = 300_000
    d2 = _unit(np.stack([rng.uniform(-0.6, 0.6, n2), rng.uniform(-0.4, 0.4, n2), rng.choice([-1.0, 1.0], n2)], axis=1)).astype(np.float32)
    o2 = rng.uniform(-20, 20, (n2, 3)).astype(np.float32)
    l2 = rng.uniform(200, 600, n2).astype(np.float32)
    do, dd, dl = _dev(o2, d2, l2)
    a = _host(gs.propagate(do, dd, dl, seed=8))
    b = _host(gs.propagate(do, dd, dl, seed=8, brute=True))
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    # vertex normals change the result: the same scene without them disagrees
    plain = pkg.Scene(_wavy_cavity(np.random.default_rng(33), with_normals=(False, False))).build()
    p = _host(plain.propagate(do, dd, dl, seed=8))
    assert not np.array_equal(p["dir"], a["dir"])


def test_smooth_scene_at_scale_bvh_equals_brute_and_filter_pipeline(smooth):
    """1e6 C3 photons on the smooth toy scene: BVH traversal == all-triangle loop, conservation, and the paper's
    pipeline (prefilter + NO_EFFICIENCY) runs on it unchanged."""
    sc, gs = smooth
    w = wl.make_config("C3", n=10_000_000)
    ids = np.arange(0, w.n, 10, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    do, dd, dl = _dev(o, d, lam)
    a = _host(gs.propagate(do, dd, dl, seed=3))
    b = _host(gs.propagate(do, dd, dl, seed=3, brute=True))
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    assert int(a["counters"][:7].sum()) == len(ids) and int(a["hitmap"].sum()) == int(a["counters"][0])
    pre = gs.prefilter(do, dd, dl, [sc.info["m_det"], sc.info["m_mir"]], seed=3)
    geo = _host(gs.propagate(pre["origins"], pre["dirs"], pre["wavelengths"], flags=opx.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"]))
    k = int(pre["n_kept"].item())
    ref = oracle.trace_mesh(sc, o[:20000], d[:20000], lam[:20000], seed=3, flags=oracle.NO_EFFICIENCY)
    kept = pre["index"][:k].cpu().numpy()
    first = kept < 20000
    for key in ("state", "pixel", "surface", "bounces"):
        assert np.array_equal(geo[key][:k][first], ref[key][kept[first]]), key


def test_vertex_normal_validation():
    sc = toy_rich_scene("c2", cells=4, smooth=True)
    sc.meshes[0]["vertex_normals"] = sc.meshes[0]["vertex_normals"].copy()
    sc.meshes[0]["vertex_normals"][3, 1] = np.nan
    with pytest.raises(pkg.OpxError) as e:
        pkg.Scene(sc)
    assert e.value.status == opx.OPX_ERR_INVALID_ARG
    # zero vertex normals == no vertex normals
    z = toy_rich_scene("c2", cells=4, smooth=True)
    z.meshes[0]["vertex_normals"] = np.zeros_like(z.meshes[0]["vertex_normals"])
    gz, gp = pkg.Scene(z).build(), pkg.Scene(toy_rich_scene("c2", cells=4)).build()
    assert gz.layout()["total_bytes"] > gp.layout()["total_bytes"]
    w = wl.make_config("C1", n=5000)
    o, d, lam = w.photon_range(0, w.n)
    a, b = _host(gz.propagate(*_dev(o, d, lam), seed=1)), _host(gp.propagate(*_dev(o, d, lam), seed=1))
    for k in a:
        assert np.array_equal(a[k], b[k]), k
