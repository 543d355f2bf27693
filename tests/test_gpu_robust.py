"""GPU parity where BVH culling could go wrong: the traversal is conservative only if no box is
culled that holds a triangle the contract test accepts.  These tests aim rays at the places where
the cheap slab / beam arithmetic and the padding of the boxes are under the most strain:

  * direction components that are exactly +0, -0 or denormal, from origins away from the coordinate origin
    (the reciprocal of the slab test is infinite there);
  * origins far outside the scene (the contract's vertex - origin rounds to ulps of the ORIGIN);
  * grazing incidence (1e-6 .. 1e-3 rad) on sliver triangles (aspect 1e4) and on very large triangles, at
    coordinates near 3000 mm, in coherent bundles (beam traversal) and mixed (per-lane walk of the binary tree);
  * bundles whose direction components straddle zero (they flip the beam's "mixed axis" handling);
  * origins lying exactly on box faces.

Bar: the product walk, the binary-tree-only walk and the GPU all-triangle loop (same arithmetic, no hierarchy)
agree bit for bit on every ray, and all agree with the CPU oracle on a sample."""
import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl
from workloads.scenes import MAT_ABSORBER, MAT_DETECTOR, MAT_MIRROR, N_LAMBDA, Scene

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KEYS_INT = ("state", "surface", "pixel", "bounces")


def _dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def _host(out):
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def _same(a, b, what):
    for k in KEYS_INT:
        bad = np.flatnonzero(a[k] != b[k])
        assert bad.size == 0, f"{what}: {bad.size} rays differ in {k}, first at {bad[:5]}"
    for k in ("pos", "dir"):
        x, y = np.asarray(a[k], np.float64), np.asarray(b[k], np.float64)
        eq = (x == y) | (np.isnan(x) & np.isnan(y))
        assert eq.all(), f"{what}: {k} differs on {int((~eq).any(axis=1).sum())} rays"


def _check(sc, gs, o, d, lam, seed, what, sample=None, brute=True):
    """product == binary walk == GPU all-triangle loop on every ray; == oracle on `sample` (all rays if None)."""
    do, dd, dl = _dev(o, d, lam)
    prod = _host(gs.propagate(do, dd, dl, seed=seed))
    binw = _host(gs.propagate(do, dd, dl, seed=seed, binary=True))
    _same(prod, binw, what + " [product vs binary walk]")
    if brute:
        bru = _host(gs.propagate(do, dd, dl, seed=seed, brute=True))
        _same(prod, bru, what + " [product vs GPU all-triangle loop]")
        assert np.array_equal(prod["hitmap"], bru["hitmap"]) and np.array_equal(prod["counters"], bru["counters"])
    idx = np.arange(len(lam)) if sample is None else sample
    # the GPU ran id_base = 0 with ids = positions in the call: the oracle takes the same ids
    ref = oracle.trace_mesh(sc, o[idx], d[idx], lam[idx], seed=seed, ids=idx.astype(np.uint64))
    _same({k: prod[k][idx] for k in KEYS_INT + ("pos", "dir")}, ref, what + " [product vs oracle]")
    return prod


@pytest.fixture(scope="module")
def toy():
    w = wl.make_config("C2", n=1)
    return w.scene, pkg.Scene(w.scene).build()


def _unit(v):
    v = np.asarray(v, np.float64)
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def test_zero_and_signed_zero_direction_components(toy):
    """with d = (0,0,1) from o = (5,2,0) the old slab test computed inf - inf = NaN for every box
    that straddles the origin's x or y and skipped it.  Axis-aligned directions, +0 / -0 / denormal components and
    directions with one exact zero, from origins spread over the volume; first as coherent calls (one direction per
    call: beam traversal and the octant-specialised walk), then shuffled together (mixed packets: generic walk)."""
    sc, gs = toy
    rng = np.random.default_rng(5)
    n = 2048
    dirs = [(0, 0, 1), (0, 0, -1), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0),
            (-0.0, 0.0, 1), (0.0, -0.0, 1), (-0.0, -0.0, 1), (-0.0, -0.0, -1), (1e-42, -1e-42, 1), (-1e-39, 1e-45, -1),
            (0, np.sin(0.3), np.cos(0.3)), (np.sin(0.2), 0, np.cos(0.2)), (-0.0, -np.sin(0.4), np.cos(0.4)),
            (np.sin(0.1), -0.0, -np.cos(0.1)), (0.6, 0.8, 0.0), (-0.6, 0.8, -0.0)]
    all_o, all_d = [], []
    for k, dv in enumerate(dirs):
        o = np.stack([rng.uniform(-380, 380, n), rng.uniform(-250, 700, n), rng.uniform(50, 1100, n)], axis=1).astype(np.float32)
        d = np.tile(np.asarray(dv, np.float32), (n, 1))          # float32(-0.0) keeps its sign
        lam = rng.uniform(200, 600, n).astype(np.float32)
        _check(sc, gs, o, d, lam, 100 + k, f"direction {dv}", brute=False)
        all_o.append(o); all_d.append(d)
    o, d = np.concatenate(all_o), np.concatenate(all_d)
    perm = rng.permutation(len(o))
    o, d = o[perm], d[perm]
    lam = rng.uniform(200, 600, len(o)).astype(np.float32)
    got = _check(sc, gs, o, d, lam, 7, "mixed zero-component directions", brute=False)
    assert (got["state"] != 6).mean() > 0.9          # the enclosure catches (nearly) everything: nothing slipped through a box


def test_origins_far_outside_the_scene(toy):
    """Origins 5, 50, 300 and 3000 scene sizes away, aimed at points of the mirror and of the detector: the contract's
    vertex - origin rounds to ulps of the origin, so accepted hits move by up to 2^-23 |origin| -- more than the padding
    of the boxes; such rays take the walk with per-ray slack (slab2_slack)."""
    sc, gs = toy
    rng = np.random.default_rng(6)
    v = sc.meshes[0]["vertices"].astype(np.float64)
    n = 3000
    for k, scale in enumerate((5.0, 50.0, 300.0, 3000.0)):
        tgt = v[rng.integers(0, len(v), n)] + rng.normal(0, 2.0, (n, 3))
        dirn = _unit(rng.normal(0, 1, (n, 3)) * [1, 1, 0.2] + [0, 0, 1.0])
        o = (tgt - dirn * scale * 1500.0).astype(np.float32)
        d = _unit(tgt - o.astype(np.float64)).astype(np.float32)
        lam = rng.uniform(200, 600, n).astype(np.float32)
        got = _check(sc, gs, o, d, lam, 40 + k, f"origins {scale} scene sizes out", brute=True)
        assert (got["state"] != 6).mean() > 0.5


def _grazing_scene(rng, centre=3000.0):
    """Slivers (aspect 1e4), mid-size and very large triangles near |coordinate| = 3000 mm; mirrors (R = 1) and absorbers."""
    sc = Scene()
    m_abs = sc.add_material(MAT_ABSORBER, np.zeros(N_LAMBDA))
    m_mir = sc.add_material(MAT_MIRROR, np.ones(N_LAMBDA))
    m_det = sc.add_material(MAT_DETECTOR, np.full(N_LAMBDA, 0.5))
    tris = []
    def add(kind, c, e1, e2, a, b):
        tris.append((kind, np.stack([c - 0.5 * a * e1, c + 0.5 * a * e1, c + b * e2])))
    for _ in range(300):          # slivers: base 100 mm, height 0.01 mm
        e1 = _unit(rng.normal(0, 1, 3)); e2 = _unit(np.cross(e1, rng.normal(0, 1, 3)))
        add(rng.integers(0, 2), centre + rng.uniform(-150, 150, 3), e1, e2, 100.0, 0.01)
    for _ in range(300):          # ordinary facets, 5 mm
        e1 = _unit(rng.normal(0, 1, 3)); e2 = _unit(np.cross(e1, rng.normal(0, 1, 3)))
        add(rng.integers(0, 2), centre + rng.uniform(-150, 150, 3), e1, e2, 5.0, 4.3)
    for _ in range(24):           # very large triangles, 1500 mm: the barycentric weights lose the most at grazing incidence
        e1 = _unit(rng.normal(0, 1, 3)); e2 = _unit(np.cross(e1, rng.normal(0, 1, 3)))
        add(rng.integers(0, 2), centre + rng.uniform(-300, 300, 3), e1, e2, 1500.0, 1300.0)
    for kind in (0, 1):
        vs = np.concatenate([t for k, t in tris if k == kind])
        sc.add_mesh("abs" if kind == 0 else "mir", vs, np.arange(len(vs)).reshape(-1, 3), m_abs if kind == 0 else m_mir)
    # a detector quad well behind everything so that reflected rays end somewhere with a pixel
    fr = sc.add_frame([centre - 2000, centre - 2000, centre + 2500.0], [1, 0, 0], [0, 1, 0], 4.0, 4.0, 1000, 1000, 0)
    q = np.float64([[centre - 2000, centre - 2000, centre + 2500], [centre + 2000, centre - 2000, centre + 2500],
                    [centre + 2000, centre + 2000, centre + 2500], [centre - 2000, centre + 2000, centre + 2500]])
    sc.add_mesh("det", q, [[0, 1, 2], [0, 2, 3]], m_det, frame=fr)
    return sc, [t for _, t in tris]


def test_grazing_incidence_slivers_and_large_triangles():
    """>= 1e6 rays in bundles of 64 (neighbours in a tile: beam traversal) at 1e-6 .. 1e-3 rad to the plane of a sliver,
    a facet or a 1500 mm triangle near |coordinate| = 3000 mm; a quarter of the bundles straddle zero in one direction
    component, a quarter start exactly on a coordinate of the target triangle's box."""
    rng = np.random.default_rng(11)
    sc, tris = _grazing_scene(rng)
    gs = pkg.Scene(sc).build()
    nb, per = 16384, 64
    k = rng.integers(0, len(tris), nb)
    T = np.stack([tris[i] for i in k])                                    # (nb, 3, 3)
    w = rng.dirichlet([1, 1, 1], nb)
    q = np.einsum("bi,bij->bj", w, T)                                      # target point on the triangle
    e1 = _unit(T[:, 1] - T[:, 0]); nrm = _unit(np.cross(T[:, 1] - T[:, 0], T[:, 2] - T[:, 0])); e2 = np.cross(nrm, e1)
    phi = rng.uniform(0, 2 * np.pi, nb)
    theta = 10 ** rng.uniform(-6, -3, nb) * rng.choice([-1.0, 1.0], nb)
    dirn = _unit(np.cos(theta)[:, None] * (np.cos(phi)[:, None] * e1 + np.sin(phi)[:, None] * e2) + np.sin(theta)[:, None] * nrm)
    L = rng.uniform(1.0, 400.0, nb)
    # bundle: 64 rays, origins jittered by <= 0.5 mm in the triangle's plane, directions by <= 2e-5
    jit = rng.uniform(-0.5, 0.5, (nb, per, 2))
    o = (q - dirn * L[:, None])[:, None, :] + jit[..., :1] * e1[:, None, :] + jit[..., 1:] * e2[:, None, :]
    d = dirn[:, None, :] + rng.normal(0, 2e-5, (nb, per, 3))
    # a quarter of the bundles: one direction component straddles zero across the lanes (exact +0 / -0 included)
    z = np.arange(nb) % 4 == 1
    ax = rng.integers(0, 3, nb)
    comp = np.linspace(-3e-8, 3e-8, per)[None, :] * rng.choice([1.0, 10.0, 1e3], nb)[:, None]
    comp[:, per // 2] = 0.0; comp[:, per // 2 + 1] = -0.0
    for a in range(3):
        sel = z & (ax == a)
        d[sel, :, a] = comp[sel]
    d = _unit(d)
    o32, d32 = o.astype(np.float32), d.astype(np.float32)
    d32[z & (ax == 0), per // 2 + 1, 0] = np.float32(-0.0)
    # another quarter: the origin sits exactly on a coordinate plane of the target's bounding box
    f = np.flatnonzero(np.arange(nb) % 4 == 2)
    a = rng.integers(0, 3, len(f))
    o32[f, :, a] = T[f][:, :, :].astype(np.float32).min(axis=1)[np.arange(len(f)), a][:, None]
    o32, d32 = o32.reshape(-1, 3), d32.reshape(-1, 3)
    lam = rng.uniform(200, 600, len(o32)).astype(np.float32)
    sample = rng.choice(len(lam), 60_000, replace=False)
    got = _check(sc, gs, o32, d32, lam, 3, "grazing incidence", sample=np.sort(sample), brute=True)
    hit = got["state"] != 6
    assert hit.mean() > 0.5                     # the rays do meet the geometry they were aimed at
    assert (got["bounces"] >= 1).mean() > 0.1   # and mirrors send a good part of them on to further segments


def test_grazing_rays_on_the_c4_scene_mirrors():
    """The same at production scale: bundles grazing the spherical-mirror facets and their backing plates (1 mm behind)
    of the 1.01e6-triangle scene; product == binary walk == GPU all-triangle loop on all 262 144 rays, == oracle on a sample."""
    w = wl.make_config("C4", n=1)
    sc = w.scene
    gs = pkg.Scene(sc).build()
    rng = np.random.default_rng(12)
    mir = [m for m in sc.meshes if sc.materials[m["material"]]["kind"] == MAT_MIRROR]
    nb, per = 4096, 64
    o_l, d_l = [], []
    for b in range(nb):
        m = mir[rng.integers(0, len(mir))]
        t = m["vertices"][m["indices"][rng.integers(0, len(m["indices"]))]].astype(np.float64)
        q = rng.dirichlet([1, 1, 1]) @ t
        e1 = _unit(t[1] - t[0]); nrm = _unit(np.cross(t[1] - t[0], t[2] - t[0])); e2 = np.cross(nrm, e1)
        phi, theta = rng.uniform(0, 2 * np.pi), 10 ** rng.uniform(-5, -2.5) * rng.choice([-1.0, 1.0])
        dirn = _unit(np.cos(theta) * (np.cos(phi) * e1 + np.sin(phi) * e2) + np.sin(theta) * nrm)
        jit = rng.uniform(-0.3, 0.3, (per, 2))
        o_l.append(q - dirn * rng.uniform(2.0, 60.0) + jit[:, :1] * e1 + jit[:, 1:] * e2)
        d_l.append(_unit(dirn + rng.normal(0, 1e-5, (per, 3))))
    o, d = np.concatenate(o_l).astype(np.float32), np.concatenate(d_l).astype(np.float32)
    lam = rng.uniform(200, 600, len(o)).astype(np.float32)
    sample = np.sort(rng.choice(len(lam), 1500, replace=False))
    _check(sc, gs, o, d, lam, 9, "grazing on C4 mirrors", sample=sample, brute=True)


def test_incoherent_packets_take_the_per_lane_walk(toy):
    """Packets of unrelated rays -- isotropic directions from origins scattered through the enclosure, in an order that puts
    no two neighbours into one packet -- are too wide for a beam: every packet-segment is walked per lane through the binary
    tree (closest_hit_own), in all four kernel shapes' size ranges; a block of coherent cone photons in the middle of the call
    makes the same tiles hold beam packets and per-lane packets side by side."""
    sc, gs = toy
    rng = np.random.default_rng(77)
    n = 160_000
    lo, hi = sc.meshes[-1]["vertices"].min(axis=0) + 5.0, sc.meshes[-1]["vertices"].max(axis=0) - 5.0
    o = (lo + (hi - lo) * rng.random((n, 3))).astype(np.float32)
    d = _unit(rng.normal(size=(n, 3))).astype(np.float32)
    lam = rng.uniform(200.0, 600.0, n).astype(np.float32)
    w = wl.make_config("C2", n=200_000)
    co, cd, cl = w.photon_range(0, 40_000)
    o[60_000:100_000], d[60_000:100_000], lam[60_000:100_000] = co, cd, cl
    sample = np.arange(0, n, 41)
    prod = _check(sc, gs, o, d, lam, 9, "incoherent rays", sample=sample)
    assert len(np.unique(prod["state"])) >= 4
    # the instrumented product kernel saw both kinds of packet-segments
    _, st = gs.propagate_packet_stats(*_dev(o, d, lam), seed=9)
    assert st["fallback_segments"] > 3000 and st["beam_segments"] > 1000
    # sizes that take the 512-photon tiles, the single wave and the large tiles
    for m in (3_000, 100_000, n):
        do, dd, dl = _dev(o[:m], d[:m], lam[:m])
        part = _host(gs.propagate(do, dd, dl, seed=9))
        for k in KEYS_INT + ("pos", "dir"):
            assert np.array_equal(part[k], prod[k][:m], equal_nan=k in ("pos", "dir")), (m, k)
