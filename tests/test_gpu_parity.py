"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle on the same seeded
inputs -- element by element.  Bar (BASELINE.json north_star): integer outputs (state, surface,
pixel, bounces, hit-map, counters) bit-exact except for at most 1e-5 of photons; positions within
1e-3 mm; directions within 1e-6 rad.  Run with `pytest -m gpu` on the B200 box."""
import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl
from workloads.scenes import MAT_ABSORBER, MAT_DETECTOR, MAT_MIRROR, N_LAMBDA, Scene

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

POS_TOL_MM, DIR_TOL_RAD, MISMATCH_FRACTION = 1e-3, 1e-6, 1e-5


def _dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def _host(out):
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


@pytest.fixture(scope="module")
def toy():
    w = wl.make_config("C2", n=1)
    return w.scene, pkg.Scene(w.scene).build()


@pytest.fixture(scope="module")
def toy_flat():
    w = wl.make_config("C1", n=1)
    return w.scene, pkg.Scene(w.scene).build()


def assert_parity(got, ref, n, check_maps=True):
    """Element-by-element comparison with the tolerances of north_star."""
    budget = max(1, int(MISMATCH_FRACTION * n)) if n else 0
    bad = np.zeros(n, dtype=bool)
    for k in ("state", "surface", "pixel", "bounces"):
        bad |= got[k] != ref[k]
    assert int(bad.sum()) <= budget, f"{int(bad.sum())} of {n} photons differ in integer outputs (budget {budget})"
    ok = ~bad
    dpos = np.abs(got["pos"].astype(np.float64) - ref["pos"])[ok]
    assert dpos.size == 0 or dpos.max() <= POS_TOL_MM, f"max |dpos| = {dpos.max()} mm"
    g, r = got["dir"].astype(np.float64)[ok], ref["dir"][ok]
    fin = np.isfinite(r).all(axis=1)
    ang = np.linalg.norm(np.cross(g[fin], r[fin]), axis=1) / np.maximum(np.linalg.norm(r[fin], axis=1) ** 2, 1e-300)
    assert ang.size == 0 or ang.max() <= DIR_TOL_RAD, f"max direction difference {ang.max()} rad"
    if check_maps:
        hm_diff = np.abs(got["hitmap"].astype(np.int64) - ref["hitmap"].astype(np.int64)).sum()
        assert hm_diff <= 2 * int(bad.sum())
        cdiff = np.abs(got["counters"][:7].astype(np.int64) - ref["counters"][:7].astype(np.int64)).sum()
        assert cdiff <= 2 * int(bad.sum())
        if not bad.any():
            assert int(got["counters"][7]) == int(ref["counters"][7])
    return int(bad.sum()), (float(dpos.max()) if dpos.size else 0.0)


# ------------------------------------------------------------------------------------ configs
def test_c1_full_parity(toy_flat):
    """Config 0 at its full size (1e5 photons) on the 20 014-triangle mesh: every photon."""
    sc, gs = toy_flat
    w = wl.make_config("C1")
    o, d, lam = w.photon_range(0, w.n)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=0))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=0)
    nbad, dmax = assert_parity(got, ref, w.n)
    assert nbad == 0 and dmax == 0.0          # same fp32 operation sequence: expected to be bit-identical
    assert np.array_equal(got["pos"].astype(np.float64), ref["pos"])
    assert np.array_equal(got["dir"].astype(np.float64), ref["dir"])
    # closed-form checks on the GPU result itself (P3, P4, P6)
    det = got["state"] <= 1
    q = got["pos"][det].astype(np.float64) - sc.info["D"]
    rad = np.hypot(q @ sc.info["du"], q @ sc.info["dv"])
    assert abs(rad.mean() - 63.52) < 0.3       # (R/2) tan(theta_c), blurred by the 8 mm facets
    cnt = got["counters"][:7]
    assert cnt.sum() == w.n and abs(cnt[0] - 22500) < 4 * 132 and cnt[6] == 0
    assert got["hitmap"].sum() == cnt[0]


@pytest.mark.parametrize("name,stride,seed", [("C2", 200, 1), ("C3", 250, 2)])
def test_c2_c3_sampled_parity(toy, name, stride, seed):
    """Configs 1 and 2 (1e7 photons): every `stride`-th id of the full workload against the oracle.
    A photon's result depends only on (scene, inputs[i], seed, id), so parity on an id subset is
    exact parity for those ids."""
    sc, gs = toy
    w = wl.make_config(name)
    ids = np.arange(0, w.n, stride, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    # ids are strided: the GPU call takes a contiguous id range, so run id_base = 0 on both sides
    got = _host(gs.propagate(*_dev(o, d, lam), seed=seed))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=seed)
    nbad, dmax = assert_parity(got, ref, len(ids))
    assert nbad == 0 and dmax == 0.0
    if name == "C3":
        assert len(np.unique(ref["state"])) >= 5        # the workload exercises the terminal states


def test_c2_bench_launch_itself_against_the_oracle(toy):
    """The launch bench.py times on C2 -- all 1e7 point-source photons, contiguous ids, one opx_propagate call (large tiles,
    packets of ring neighbours) -- compared with the oracle on every 4000th of its records (the oracle traces those ids alone:
    a photon's result depends on (scene, inputs[i], seed, id) only), plus the size-independent properties on all of them."""
    sc, gs = toy
    w = wl.make_config("C2")
    pin = [torch.empty((w.n, 3), dtype=torch.float32), torch.empty((w.n, 3), dtype=torch.float32), torch.empty(w.n, dtype=torch.float32)]
    for a in range(0, w.n, 2_000_000):
        for dst, src in zip(pin, w.photon_range(a, a + 2_000_000)):
            dst[a:a + 2_000_000] = torch.from_numpy(src)
    got = gs.propagate(*(x.cuda() for x in pin), seed=0)
    torch.cuda.synchronize()
    ids = np.arange(0, w.n, 4000, dtype=np.uint64)
    idx = torch.from_numpy(ids.astype(np.int64)).cuda()
    sub = {k: got[k][idx].cpu().numpy() for k in ("state", "pixel", "surface", "bounces", "pos", "dir")}
    o, d, lam = w.photons(ids)
    ref = oracle.trace_mesh(sc, o, d, lam, seed=0, ids=ids)
    for k in ("state", "pixel", "surface", "bounces"):
        assert np.array_equal(sub[k], ref[k]), k
    assert np.array_equal(sub["pos"].astype(np.float64), ref["pos"]) and np.array_equal(sub["dir"].astype(np.float64), ref["dir"])
    cnt = got["counters"].cpu().numpy()
    assert cnt[:7].sum() == w.n and int(got["hitmap"].sum().item()) == cnt[0]
    det = got["state"] == 0
    assert torch.equal(torch.bincount(got["pixel"][det].long(), minlength=gs.n_pixels).int(), got["hitmap"].int())
    assert bool((got["pixel"][~(det | (got["state"] == 1))] == -1).all())


def test_both_cta_shapes_against_the_oracle(toy):
    """opx_propagate picks 512-photon tiles (one packet per warp) for small calls (on this scene: up to 75 776 photons), a single
    wave of 1024-thread CTAs from there to 151 552 photons, and large tiles (512 threads x 4 photons)
    above: 620 000 contiguous C3 photons take the large tiles, their first 50 000 alone the small ones, their first
    120 000 the single wave; all must reproduce the oracle, hence each other, bit for bit.  (The 512-thread
    shape is pinned by test_no_efficiency_trace_at_scale on this scene and by tests/test_gpu_filter.py on the large one.)"""
    sc, gs = toy
    w = wl.make_config("C3", n=2_000_000)
    n = 620_000
    o, d, lam = w.photon_range(700_000, 700_000 + n)
    do, dd, dl = _dev(o, d, lam)
    big = _host(gs.propagate(do, dd, dl, seed=21, photon_id_base=700_000))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=21, id_base=700_000)
    nbad, dmax = assert_parity(big, ref, n)
    assert nbad == 0 and dmax == 0.0
    m = 50_000
    small = _host(gs.propagate(do[:m].contiguous(), dd[:m].contiguous(), dl[:m].contiguous(), seed=21, photon_id_base=700_000))
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(small[k], big[k][:m]), k
    m = 120_000
    wave = gs.propagate(do[:m].contiguous(), dd[:m].contiguous(), dl[:m].contiguous(), seed=21, photon_id_base=700_000)
    assert pkg.last_kernel() == "k_propagate_packet<1024, 1, 1, 0>"
    wave = _host(wave)
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(wave[k], big[k][:m]), k


def test_propagate_is_cuda_graph_capturable(toy):
    """opx_propagate performs stream operations only (kernel attributes are set at opx_bvh_build): a call captured into a CUDA
    graph and replayed gives the records of the plain call."""
    sc, gs = toy
    w = wl.make_config("C3", n=300_000)
    do, dd, dl = _dev(*w.photon_range(0, 200_000))
    plain = _host(gs.propagate(do, dd, dl, seed=3))
    rec = gs.alloc_records(200_000)
    hm, ct = gs.alloc_accumulators()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        g.capture_begin()
        gs.propagate(do, dd, dl, seed=3, records=rec, hitmap=hm, counters=ct, stream=side)
        g.capture_end()
    for _ in range(2):
        hm.zero_(); ct.zero_(); rec["state"].fill_(99)
        g.replay()
    torch.cuda.synchronize()
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(rec[k].cpu().numpy(), plain[k]), k
    assert np.array_equal(hm[:gs.n_pixels].cpu().numpy(), plain["hitmap"]) and np.array_equal(ct.cpu().numpy(), plain["counters"])


def test_id_base_and_chunking(toy):
    """Global photon id = base + i keys the RNG: chunked calls reproduce the one-shot call, and match
    the oracle run with the same ids."""
    sc, gs = toy
    w = wl.make_config("C3", n=2_000_000)
    o, d, lam = w.photon_range(1_000_000, 1_030_000)
    do, dd, dl = _dev(o, d, lam)
    whole = _host(gs.propagate(do, dd, dl, seed=5, photon_id_base=1_000_000))
    hm, ct = gs.alloc_accumulators()
    parts = []
    for a, b in ((0, 7), (7, 10_001), (10_001, 30_000)):
        parts.append(_host(gs.propagate(do[a:b].contiguous(), dd[a:b].contiguous(), dl[a:b].contiguous(), seed=5,
                                        photon_id_base=1_000_000 + a, hitmap=hm, counters=ct)))
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), whole[k]), k
    assert np.array_equal(parts[-1]["hitmap"], whole["hitmap"]) and np.array_equal(parts[-1]["counters"], whole["counters"])
    ref = oracle.trace_mesh(sc, o[:5000], d[:5000], lam[:5000], seed=5, id_base=1_000_000)
    assert np.array_equal(whole["state"][:5000], ref["state"]) and np.array_equal(whole["pixel"][:5000], ref["pixel"])
    other = _host(gs.propagate(do, dd, dl, seed=5, photon_id_base=0))
    assert not np.array_equal(other["state"], whole["state"])       # different ids => different draws
    # 64-bit ids: the high word reaches the generator
    hi = _host(gs.propagate(do[:2000].contiguous(), dd[:2000].contiguous(), dl[:2000].contiguous(), seed=5, photon_id_base=(1 << 40)))
    ref_hi = oracle.trace_mesh(sc, o[:2000], d[:2000], lam[:2000], seed=5, id_base=(1 << 40))
    assert np.array_equal(hi["state"], ref_hi["state"])
    big_seed = (0xDEADBEEF << 32) | 0x12345678
    hs = _host(gs.propagate(do[:2000].contiguous(), dd[:2000].contiguous(), dl[:2000].contiguous(), seed=big_seed))
    ref_hs = oracle.trace_mesh(sc, o[:2000], d[:2000], lam[:2000], seed=big_seed)
    assert np.array_equal(hs["state"], ref_hs["state"])


def test_bvh_equals_gpu_brute_force_at_scale(toy):
    """1e6 photons of C3: BVH traversal and the all-triangle GPU loop agree on every output
    (separates the BVH from the arithmetic contract), plus determinism and conservation (P4)."""
    sc, gs = toy
    w = wl.make_config("C3", n=10_000_000)
    ids = np.arange(0, w.n, 10, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    do, dd, dl = _dev(o, d, lam)
    a = _host(gs.propagate(do, dd, dl, seed=3))
    b = _host(gs.propagate(do, dd, dl, seed=3, brute=True))
    c = _host(gs.propagate(do, dd, dl, seed=3))
    for k in a:
        assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a[k], c[k]), k            # two runs are byte-identical
    n = len(ids)
    assert a["counters"][:7].sum() == n
    assert np.array_equal(a["counters"][:7], np.bincount(a["state"], minlength=7))
    det = a["state"] == 0
    assert np.array_equal(a["hitmap"], np.bincount(a["pixel"][det], minlength=gs.n_pixels))
    assert a["counters"][7] == (a["bounces"].astype(np.int64) + (a["state"] != 5)).sum()
    assert np.all(a["pixel"][a["state"] > 1] == -1) and np.all(a["surface"][a["state"] == 6] == -1)


# ------------------------------------------------------------------------- BVH invariants (P14)
@pytest.fixture(scope="module")
def lhcb():
    sc = wl.lhcb_like_scene()
    return sc, pkg.Scene(sc).build()


def _check_lbvh(sc, gs):
    lay, T = gs.layout(), gs.n_triangles
    ws = gs.workspace
    base = (ws.data_ptr() + 255) // 256 * 256 - ws.data_ptr()
    raw = ws.cpu().numpy()[base:]
    keys = raw[lay["sorted_keys"]:lay["sorted_keys"] + 8 * T].view(np.uint64)
    assert np.all(keys[1:] >= keys[:-1])                                      # sorted 63-bit Morton keys
    tris = raw[lay["triangles"]:lay["triangles"] + 48 * T].view(np.float32).reshape(T, 3, 4)
    gid = tris[:, 0, 3].view(np.int32)
    assert np.array_equal(np.sort(gid), np.arange(T))                          # a permutation: each triangle in one leaf
    flat, surf = sc.flat_triangles()
    assert np.array_equal(tris[:, :, :3], flat[gid])                           # vertices carried unchanged
    assert np.array_equal(tris[:, 1, 3].view(np.int32), surf[gid])
    nodes = raw[lay["nodes"]:lay["nodes"] + 64 * (T - 1)].view(np.float32).reshape(T - 1, 16)
    child = nodes[:, 12:14].view(np.int32)
    parents = raw[lay["parents"]:lay["parents"] + 4 * (2 * T - 1)].view(np.int32)
    assert parents[0] == -1 and np.all(parents[1:T - 1] >= 0) and np.all(parents[T - 1:] >= 0)
    internal = child[child >= 0]
    leaves = ~child[child < 0]
    assert np.array_equal(np.sort(internal), np.arange(1, T - 1))              # every internal node but the root has one parent
    assert np.array_equal(np.sort(leaves), np.arange(T))                       # every leaf referenced exactly once
    # every child box contains the boxes / triangles below it (all nodes at once)
    lo = np.stack([nodes[:, 0:3], nodes[:, 6:9]], axis=1)                      # (node, child, xyz)
    hi = np.stack([nodes[:, 3:6], nodes[:, 9:12]], axis=1)
    tlo, thi = tris[:, :, :3].min(axis=1), tris[:, :, :3].max(axis=1)
    for c in range(2):
        r = child[:, c]
        inner, leaf = r >= 0, r < 0
        assert np.all(lo[inner, c] <= lo[r[inner]].min(axis=1)) and np.all(hi[inner, c] >= hi[r[inner]].max(axis=1))
        assert np.all(lo[leaf, c] < tlo[~r[leaf]]) and np.all(hi[leaf, c] > thi[~r[leaf]])   # padded: strict
    # the parent array agrees with the child links, and every leaf reaches the root
    pc = parents[1:T - 1]
    assert np.all((child[pc, 0] == np.arange(1, T - 1)) | (child[pc, 1] == np.arange(1, T - 1)))
    pl = parents[T - 1:]
    assert np.all((child[pl, 0] == ~np.arange(T)) | (child[pl, 1] == ~np.arange(T)))
    cur, depth = pl.copy(), np.ones(T, np.int64)
    while np.any(cur > 0):
        live = cur > 0
        cur[live] = parents[cur[live]]
        depth[live] += 1
        assert depth.max() <= 96                      # depth bound the traversal stacks are sized for
    return int(depth.max())


def test_p14_lbvh_invariants(toy):
    sc, gs = toy
    assert _check_lbvh(sc, gs) < 40


def test_c4_scene_bvh_and_sampled_parity(lhcb):
    """Config 3: LHCb-RICH1-like scene, 1 010 060 triangles, 64 000 pixels in 1000 frames.  BVH
    invariants, parity with the oracle on every 50 000th photon id of the 1e8-photon workload, and
    BVH traversal == GPU all-triangle loop on 30 000 more."""
    sc, gs = lhcb
    assert abs(gs.n_triangles - 1_000_000) < 50_000 and gs.n_pixels == 64_000
    assert _check_lbvh(sc, gs) <= 96
    w = wl.make_config("C4")
    ids = np.arange(0, w.n, 50_000, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=6))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=6)
    nbad, dmax = assert_parity(got, ref, len(ids))
    assert nbad == 0 and dmax == 0.0
    assert len(np.unique(ref["state"])) >= 5 and ref["bounces"].max() == 2
    assert 0.4 < np.mean(ref["bounces"] == 2) < 0.9          # most photons take the two-mirror path
    ids2 = np.arange(7, w.n, 3_333, dtype=np.uint64)[:30_000]
    o, d, lam = w.photons(ids2)
    do, dd, dl = _dev(o, d, lam)
    a = _host(gs.propagate(do, dd, dl, seed=6))
    b = _host(gs.propagate(do, dd, dl, seed=6, brute=True))
    for k in a:
        assert np.array_equal(a[k], b[k], equal_nan=True) if a[k].dtype.kind == "f" else np.array_equal(a[k], b[k]), k
    assert a["counters"][:7].sum() == len(ids2) and a["hitmap"].sum() == a["counters"][0]


def test_c4_bench_launch_itself_against_the_oracle(lhcb):
    """The launch bench.py's headline times -- all 1e8 track photons of C4, contiguous ids, ONE opx_propagate call on the
    1.01e6-triangle scene -- against the oracle on every 250 000th of its records (the oracle traces those ids alone), plus the
    size-independent properties on all 1e8; the detected-only form of the same launch lists exactly the DETECTED records."""
    import concurrent.futures
    sc, gs = lhcb
    w = wl.make_config("C4")
    n = w.n
    pin = [torch.empty((n, 3), dtype=torch.float32), torch.empty((n, 3), dtype=torch.float32), torch.empty(n, dtype=torch.float32)]
    step = 2_000_000

    def fill(a):
        for dst, src in zip(pin, w.photon_range(a, min(n, a + step))):
            dst[a:a + step] = torch.from_numpy(src)
    with concurrent.futures.ThreadPoolExecutor(max_workers=8) as ex:
        list(ex.map(fill, range(0, n, step)))
    do, dd, dl = (x.cuda() for x in pin)
    got = gs.propagate(do, dd, dl, seed=0)
    assert pkg.last_kernel() == "k_propagate_packet<512, 4, 2, 0>"
    torch.cuda.synchronize()
    ids = np.arange(11, n, 250_000, dtype=np.uint64)
    idx = torch.from_numpy(ids.astype(np.int64)).cuda()
    sub = {k: got[k][idx].cpu().numpy() for k in ("state", "pixel", "surface", "bounces", "pos", "dir")}
    o, d, lam = w.photons(ids)
    ref = oracle.trace_mesh(sc, o, d, lam, seed=0, ids=ids)
    for k in ("state", "pixel", "surface", "bounces"):
        assert np.array_equal(sub[k], ref[k]), k
    assert np.array_equal(sub["pos"].astype(np.float64), ref["pos"]) and np.array_equal(sub["dir"].astype(np.float64), ref["dir"])
    cnt = got["counters"].cpu().numpy()
    assert cnt[:7].sum() == n and int(got["hitmap"].long().sum().item()) == cnt[0]
    det = got["state"] == 0
    assert torch.equal(torch.bincount(got["pixel"][det].long(), minlength=gs.n_pixels).int(), got["hitmap"].int())
    lst = gs.propagate_detected(do, dd, dl, seed=0, capacity=int(cnt[0]) + 16)
    torch.cuda.synchronize()
    k = int(lst["n_detected"].item())
    assert k == cnt[0] and torch.equal(lst["id"][:k], torch.nonzero(det).flatten())
    assert torch.equal(lst["pos"][:k], got["pos"][det]) and torch.equal(lst["pixel"][:k], got["pixel"][det])


def test_c5_sampled_parity(lhcb):
    """Config 4 (the stress config): every 500 000th photon id of the 1e9-photon workload of mixed tracks
    (beta in [0.9999, 1], origins in a 200 mm disc) on the C4 scene against the oracle, through a chunked call
    sequence with advancing id bases as the config streams it."""
    sc, gs = lhcb
    w = wl.make_config("C5")
    ids = np.arange(3, w.n, 500_000, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    ref = oracle.trace_mesh(sc, o, d, lam, seed=9)
    do, dd, dl = _dev(o, d, lam)
    hm, ct = gs.alloc_accumulators()
    parts = []
    for a, b in ((0, 700), (700, 701), (701, len(ids))):
        parts.append(_host(gs.propagate(do[a:b].contiguous(), dd[a:b].contiguous(), dl[a:b].contiguous(), seed=9,
                                        photon_id_base=a, hitmap=hm, counters=ct)))
    got = {k: np.concatenate([p[k] for p in parts]) for k in ("state", "surface", "pixel", "bounces", "pos", "dir")}
    got["hitmap"], got["counters"] = parts[-1]["hitmap"], parts[-1]["counters"]
    nbad, dmax = assert_parity(got, ref, len(ids))
    assert nbad == 0 and dmax == 0.0
    assert len(np.unique(ref["state"])) >= 5 and ref["bounces"].max() == 2


def test_rebuild_is_deterministic(toy):
    sc, _ = toy
    a = pkg.Scene(sc).build()
    b = pkg.Scene(sc).build()
    lay, T = a.layout(), a.n_triangles
    ba = (a.workspace.data_ptr() + 255) // 256 * 256 - a.workspace.data_ptr()
    bb = (b.workspace.data_ptr() + 255) // 256 * 256 - b.workspace.data_ptr()
    used = dict(nodes=64 * (T - 1), triangles=48 * T, normals=16 * T, surfaces=8 * a.n_surfaces,
                tables=4 * 3 * N_LAMBDA, frames=64, sorted_keys=8 * T, parents=4 * (2 * T - 1))
    for k, nbytes in used.items():                # the alignment gaps between the arrays are never written
        off = lay[k]
        assert torch.equal(a.workspace[ba + off:ba + off + nbytes], b.workspace[bb + off:bb + off + nbytes]), k


# ----------------------------------------------------------------------------------- edge cases
def test_edge_cases_empty_nan_escape(toy):
    sc, gs = toy
    z3, z1 = torch.zeros((0, 3), device="cuda"), torch.zeros(0, device="cuda")
    out = _host(gs.propagate(z3, z3, z1))
    assert out["state"].size == 0 and out["hitmap"].sum() == 0 and out["counters"].sum() == 0
    nob = wl.toy_rich_scene(cells=4, enclosure=False)
    g2 = pkg.Scene(nob).build()
    o = np.zeros((5, 3), np.float32)
    d = np.float32([[np.nan, 0, 1], [0, 0, 0], [0, 0, -1], [0, 0, 1], [np.inf, 0, 1]])
    lam = np.float32([400, 400, 400, np.nan, 1e9])
    got = _host(g2.propagate(*_dev(o, d, lam), seed=0))
    ref = oracle.trace_mesh(nob, o, d, lam, seed=0)
    assert list(got["state"][:3]) == [6, 6, 6] and np.all(got["surface"][:3] == -1) and np.all(got["pos"][:3] == 0)
    for k in ("state", "surface", "pixel", "bounces"):
        assert np.array_equal(got[k], ref[k]), k
    assert np.array_equal(np.isnan(got["dir"]), np.isnan(ref["dir"]))


def test_tiny_scenes():
    """0, 1 and 2 triangles (no hierarchy / a single node)."""
    rng = np.random.default_rng(0)
    n = 2000
    d = np.stack([rng.uniform(-0.3, 0.3, n), rng.uniform(-0.3, 0.3, n), np.ones(n)], axis=1)
    d = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    o = np.zeros((n, 3), np.float32)
    lam = rng.uniform(200, 600, n).astype(np.float32)
    for ntri in (0, 1, 2):
        sc = Scene()
        m = sc.add_material(MAT_DETECTOR, np.full(N_LAMBDA, 0.5))
        fr = sc.add_frame([-50, -50, 100.0], [1, 0, 0], [0, 1, 0], 1.0, 1.0, 100, 100, 0)
        if ntri:
            sc.add_mesh("d", [[-50, -50, 100.0], [50, -50, 100.0], [50, 50, 100.0], [-50, 50, 100.0]],
                        [[0, 1, 2], [0, 2, 3]][:ntri], m, frame=fr)
        gs = pkg.Scene(sc).build()
        got = _host(gs.propagate(*_dev(o, d, lam), seed=4))
        ref = oracle.trace_mesh(sc, o, d, lam, seed=4)
        assert_parity(got, ref, n)
        assert (got["state"] == 6).sum() == (n if ntri == 0 else (ref["state"] == 6).sum())


def test_bounce_limit_and_duplicate_keys():
    """Two parallel mirrors (triangles of a quad share an AABB centre => equal Morton keys)."""
    sc = Scene()
    m = sc.add_material(MAT_MIRROR, np.ones(N_LAMBDA))
    for z in (-10.0, 10.0):
        sc.add_mesh("m", [[-50, -50, z], [50, -50, z], [50, 50, z], [-50, 50, z]], [[0, 1, 2], [0, 2, 3]], m)
    gs = pkg.Scene(sc).build()
    o = np.zeros((64, 3), np.float32)
    d = np.tile(np.float32([0.01, 0.003, 1.0]), (64, 1))
    d[:, 0] += np.linspace(0, 0.02, 64, dtype=np.float32)
    lam = np.full(64, 300.0, np.float32)
    got = _host(gs.propagate(*_dev(o, d, lam)))
    ref = oracle.trace_mesh(sc, o, d, lam)
    assert np.all(got["state"] == 5) and np.all(got["bounces"] == 16)
    assert_parity(got, ref, 64)
    assert got["counters"][7] == 64 * 16


def test_shared_edges_and_vertices_are_watertight(toy_flat):
    """Photons aimed exactly at mesh vertices and along mesh edges of the mirror: the GPU picks the
    same facet as the oracle (tie-break on global id) and none falls through."""
    sc, gs = toy_flat
    v = sc.meshes[0]["vertices"].astype(np.float64)
    rng = np.random.default_rng(1)
    ii, jj = np.meshgrid(np.arange(2, 99), np.arange(2, 99))             # interior vertices of the 101x101 grid
    pick = rng.choice((jj * 101 + ii).ravel(), 4000, replace=False)
    tgt = v[pick]
    tgt[2000:] = 0.5 * (tgt[2000:] + v[np.minimum(pick[2000:] + 1, len(v) - 1)])     # edge midpoints
    d = (tgt / np.linalg.norm(tgt, axis=1, keepdims=True)).astype(np.float32)
    o = np.zeros_like(d)
    lam = np.full(len(d), 450.0, np.float32)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=2))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=2)
    assert_parity(got, ref, len(d))
    # nothing falls through the mesh: the first interaction of every photon is on the mirror
    for r in (got, ref):
        assert np.all((r["bounces"] >= 1) | (r["state"] == 3))


# -------------------------------------------------------------------------- host path, errors
def test_propagate_host_matches_device_path(toy):
    sc, gs = toy
    w = wl.make_config("C3", n=3_000_000)
    o, d, lam = w.photon_range(2_000_000, 2_100_000)
    dev = _host(gs.propagate(*_dev(o, d, lam), seed=8, photon_id_base=2_000_000))
    pin = [torch.from_numpy(x).pin_memory() for x in (o, d, lam)]
    for chunk in (100_000, 33_333, 1 << 21):
        host = gs.propagate_host(*pin, seed=8, photon_id_base=2_000_000, chunk=chunk)
        for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
            assert np.array_equal(host[k].numpy(), dev[k]), (k, chunk)
        assert np.array_equal(host["hitmap"].numpy()[:gs.n_pixels], dev["hitmap"])
        assert np.array_equal(host["counters"].numpy(), dev["counters"])


def test_error_paths(toy):
    import ctypes as C
    from paper_2309_12496_b200 import opx
    sc, gs = toy
    lib = pkg.load_library()
    fresh = pkg.Scene(sc)
    x = torch.zeros((4, 3), device="cuda")
    with pytest.raises(pkg.OpxError) as e:
        fresh.propagate(x, x, torch.zeros(4, device="cuda"))
    assert e.value.status == opx.OPX_ERR_BAD_STATE
    scene_b, tmp_b = fresh.workspace_bytes()
    buf = torch.empty(scene_b + tmp_b + 512, dtype=torch.uint8, device="cuda")
    p = (buf.data_ptr() + 255) // 256 * 256
    assert lib.opx_bvh_build(fresh._h, C.c_void_p(p), scene_b - 1, C.c_void_p(p + scene_b), tmp_b, None) == opx.OPX_ERR_WORKSPACE_TOO_SMALL
    assert lib.opx_bvh_build(fresh._h, C.c_void_p(p + 4), scene_b, C.c_void_p(p + scene_b), tmp_b, None) == opx.OPX_ERR_INVALID_ARG
    assert lib.opx_bvh_build(fresh._h, None, scene_b, C.c_void_p(p), tmp_b, None) == opx.OPX_ERR_INVALID_ARG
    h = opx.Hits()
    assert lib.opx_propagate(gs._h, 4, 0, C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()), 0,
                             C.byref(h), None, None, None) == opx.OPX_ERR_INVALID_ARG
    with pytest.raises(pkg.OpxError):
        gs.propagate(x.cpu(), x, torch.zeros(4, device="cuda"))
    # the library still works after the refused calls
    out = _host(gs.propagate(x, x, torch.zeros(4, device="cuda")))
    assert np.all(out["state"] == 6)
    assert pkg.launch_count() > 0
