"""GPU parity for SURVEY.md 8(f) rows f1/f2: the paper's pre-propagation efficiency filter,
histogram tables, and the trace with efficiencies switched off -- opx_prefilter and
opx_propagate_flags through the C ABI against oracle.prefilter / oracle.trace_mesh(flags=NO_EFFICIENCY) on the
same seeded inputs.  Everything here is integer or a copy of input bits: the bar is bit-exact."""
import ctypes as C

import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl
from paper_2309_12496_b200 import opx
from workloads.scenes import MAT_DETECTOR, MAT_MIRROR, TABLE_HISTOGRAM, TABLE_LINEAR, Scene, toy_rich_scene

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

REC = ("state", "surface", "pixel", "bounces")


def _dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def _host(out):
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items() if k != "workspace"}


@pytest.fixture(scope="module")
def toy():
    w = wl.make_config("C2", n=1)
    return w.scene, pkg.Scene(w.scene).build()


@pytest.fixture(scope="module")
def toy_hist():
    sc = toy_rich_scene("paper_hist")
    return sc, pkg.Scene(sc).build()


@pytest.fixture(scope="module")
def lhcb():
    sc = wl.lhcb_like_scene()
    return sc, pkg.Scene(sc).build()


def _assert_records_equal(got, ref, n):
    for k in REC:
        assert np.array_equal(got[k][:n], ref[k]), k
    assert np.array_equal(got["pos"][:n].astype(np.float64), ref["pos"])
    assert np.array_equal(got["dir"][:n].astype(np.float64), ref["dir"], equal_nan=True)


# ------------------------------------------------------------------------- f2: histogram tables
def test_histogram_tables_in_flight_parity(toy_hist):
    """The paper's 33 nm / 25 nm histogram tables (400 bins of 1 nm) on the full toy mesh, drawn in flight;
    wavelengths include bin edges, both ends, values outside the table and NaN."""
    sc, gs = toy_hist
    w = wl.make_config("C1", n=20_000)
    o, d, lam = w.photon_range(0, w.n)
    lam = lam.copy()
    lam[:12] = np.float32([200, 199.999, 600, 600.001, 1e9, -5, np.nan, 233, 232.99998, 225, 575, 599.99997])
    got = _host(gs.propagate(*_dev(o, d, lam), seed=11))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=11)
    _assert_records_equal(got, ref, w.n)
    assert np.array_equal(got["hitmap"], ref["hitmap"]) and np.array_equal(got["counters"].astype(np.uint64), ref["counters"])
    assert len(np.unique(ref["state"])) >= 3


def test_mixed_table_forms_in_one_scene():
    """A linear mirror table and a histogram detector table in the same scene: each material keeps its own form."""
    rng = np.random.default_rng(3)
    sc = Scene()
    sc.n_lambda = 17
    m_mir = sc.add_material(MAT_MIRROR, rng.uniform(0.3, 1.0, 17), TABLE_LINEAR)
    m_det = sc.add_material(MAT_DETECTOR, rng.uniform(0.1, 0.9, 17), TABLE_HISTOGRAM)
    fr = sc.add_frame([-200, -200, -50.0], [1, 0, 0], [0, 1, 0], 4.0, 4.0, 100, 100, 0)
    sc.add_mesh("mirror", [[-300, -300, 100.0], [300, -300, 100.0], [300, 300, 100.0], [-300, 300, 100.0]], [[0, 1, 2], [0, 2, 3]], m_mir)
    sc.add_mesh("det", [[-200, -200, -50.0], [200, -200, -50.0], [200, 200, -50.0], [-200, 200, -50.0]], [[0, 1, 2], [0, 2, 3]], m_det, frame=fr)
    gs = pkg.Scene(sc).build()
    n = 50_000
    d = np.stack([rng.uniform(-0.5, 0.5, n), rng.uniform(-0.5, 0.5, n), np.ones(n)], axis=1)
    d = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
    o = np.zeros((n, 3), np.float32)
    lam = rng.uniform(150, 650, n).astype(np.float32)
    got = _host(gs.propagate(*_dev(o, d, lam), seed=2))
    ref = oracle.trace_mesh(sc, o, d, lam, seed=2)
    _assert_records_equal(got, ref, n)
    assert (ref["state"] == 0).sum() > 1000 and (ref["state"] == 1).sum() > 1000 and (ref["state"] == 3).sum() > 1000
    # the filter sees the same forms
    f = oracle.prefilter(sc, lam, [m_det, m_mir], seed=2)
    out = _host(gs.prefilter(*_dev(o, d, lam), [m_det, m_mir], seed=2))
    assert int(out["n_kept"][0]) == len(f.index) and np.array_equal(out["index"][:len(f.index)].view(np.uint32), f.index)


# -------------------------------------------------------------------------- f1: the filter itself
@pytest.mark.parametrize("n,id_base", [(1, 0), (31, 5), (2048, 0), (2049, 1 << 40), (1_000_037, 123_456_789)])
def test_prefilter_matches_oracle(toy, n, id_base):
    """Keep decisions, their order (stable compaction) and the copied photon bits, on sizes around the 32-photon
    mask word and the 2048-photon block and on ~490 blocks with a ragged tail; 64-bit ids reach the generator."""
    sc, gs = toy
    w = wl.make_config("C3", n=max(n, 2))
    o, d, lam = w.photon_range(0, n)
    fac = [sc.info["m_det"], sc.info["m_mir"], sc.info["m_mir"]]          # "the three efficiencies"
    f = oracle.prefilter(sc, lam, fac, seed=9, id_base=id_base)
    out = _host(gs.prefilter(*_dev(o, d, lam), fac, seed=9, photon_id_base=id_base))
    k = len(f.index)
    assert int(out["n_kept"][0]) == k
    assert np.array_equal(out["index"][:k].view(np.uint32), f.index)
    assert np.array_equal(out["origins"][:k], o[f.index]) and np.array_equal(out["dirs"][:k], d[f.index])
    assert np.array_equal(out["wavelengths"][:k].view(np.uint32), lam[f.index].view(np.uint32))
    if n > 10_000:
        assert 0.05 < k / n < 0.35 and np.all(np.diff(f.index.astype(np.int64)) > 0)


def test_prefilter_degenerate_cases(toy):
    sc, gs = toy
    w = wl.make_config("C3", n=5000)
    o, d, lam = w.photon_range(0, 5000)
    do, dd, dl = _dev(o, d, lam)
    # no factors: everything is kept, in order
    out = _host(gs.prefilter(do, dd, dl, [], seed=1))
    assert int(out["n_kept"][0]) == 5000 and np.array_equal(out["index"], np.arange(5000, dtype=np.int32))
    assert np.array_equal(out["origins"], o) and np.array_equal(out["wavelengths"], lam)
    # no photons: the count is overwritten with 0
    z3, z1 = torch.zeros((0, 3), device="cuda"), torch.zeros(0, device="cuda")
    pre = dict(origins=z3.clone(), dirs=z3.clone(), wavelengths=z1.clone(), index=torch.zeros(0, dtype=torch.int32, device="cuda"),
               n_kept=torch.full((1,), 77, dtype=torch.int64, device="cuda"))
    assert int(_host(gs.prefilter(z3, z3, z1, [sc.info["m_det"]], out=pre))["n_kept"][0]) == 0
    # NaN wavelength: bin/segment 0 of the table, as the oracle; the same material eight times
    lam2 = lam.copy()
    lam2[::7] = np.nan
    fac = [sc.info["m_mir"]] * 8
    f = oracle.prefilter(sc, lam2, fac, seed=3)
    out = _host(gs.prefilter(do, dd, torch.from_numpy(lam2).cuda(), fac, seed=3))
    assert int(out["n_kept"][0]) == len(f.index) and np.array_equal(out["index"][:len(f.index)].view(np.uint32), f.index)
    # a second call reuses the same output buffers and overwrites the count
    again = gs.prefilter(do, dd, dl, [sc.info["m_det"]], seed=1)
    k1 = int(again["n_kept"].item())
    again = gs.prefilter(do, dd, dl, [sc.info["m_det"], sc.info["m_mir"]], seed=1, out=again)
    assert 0 < int(again["n_kept"].item()) <= k1


# --------------------------------------------------------------- f1: filter, then trace survivors
def test_filter_then_trace_matches_oracle_c4(lhcb):
    """The paper's pipeline on the C4 scene: filter on QE x R x R, then trace the survivors with efficiencies off,
    the survivor count staying on the device (no host round trip between the two calls)."""
    sc, gs = lhcb
    w = wl.make_config("C4")
    ids = np.arange(11, w.n, 10_000, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    n = len(ids)
    m_mir = next(i for i, m in enumerate(sc.materials) if m["kind"] == MAT_MIRROR)
    m_det = next(i for i, m in enumerate(sc.materials) if m["kind"] == MAT_DETECTOR)
    fac = [m_det, m_mir, m_mir]
    f = oracle.prefilter(sc, lam, fac, seed=6)
    k = len(f.index)
    ref = oracle.trace_mesh(sc, o[f.index], d[f.index], lam[f.index], seed=6, flags=oracle.NO_EFFICIENCY)
    pre = gs.prefilter(*_dev(o, d, lam), fac, seed=6)
    rec = gs.alloc_records(n)
    for t in rec.values():
        t.fill_(113)                                              # sentinel: records beyond n_kept stay untouched
    got = _host(gs.propagate(pre["origins"], pre["dirs"], pre["wavelengths"], seed=6, records=rec,
                             flags=opx.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"]))
    assert int(pre["n_kept"].item()) == k and 0.05 < k / n < 0.35
    _assert_records_equal(got, ref, k)
    assert np.array_equal(got["hitmap"], ref["hitmap"]) and np.array_equal(got["counters"].astype(np.uint64), ref["counters"])
    assert int(got["counters"][:7].sum()) == k
    assert np.all(got["state"][k:] == 113) and np.all(got["pixel"][k:] == 113) and np.all(got["bounces"][k:] == 113)
    # 8x8 pixels of 2.88 mm fill 13 % of a 64 mm module (R10): most two-mirror photons end DETECTOR_DEAD
    assert not np.isin(ref["state"], [1, 3]).any() and (ref["state"] == 0).sum() > 0.05 * k
    assert np.isin(ref["state"], [0, 4]).sum() > 0.4 * k and ref["bounces"].max() == 2


def test_no_efficiency_trace_at_scale(toy):
    """1e6 C3 photons: the NO_EFFICIENCY trace ignores seed and ids, never rejects, agrees with the GPU all-triangle
    loop's geometry, and an in-flight DETECTED photon keeps its record (same path)."""
    sc, gs = toy
    w = wl.make_config("C3", n=10_000_000)
    ids = np.arange(0, w.n, 10, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    do, dd, dl = _dev(o, d, lam)
    a = _host(gs.propagate(do, dd, dl, seed=1, flags=opx.FLAG_NO_EFFICIENCY))
    b = _host(gs.propagate(do, dd, dl, seed=99, photon_id_base=12345, flags=opx.FLAG_NO_EFFICIENCY))
    c = _host(gs.propagate(do, dd, dl, seed=1))
    for key in a:
        assert np.array_equal(a[key], b[key], equal_nan=True) if a[key].dtype.kind == "f" else np.array_equal(a[key], b[key]), key
    assert not np.isin(a["state"], [1, 3]).any() and int(a["counters"][:7].sum()) == len(ids)
    det = c["state"] == 0
    assert det.sum() > 1000
    for key in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(a[key][det], c[key][det]), key
    ref = oracle.trace_mesh(sc, o[:3000], d[:3000], lam[:3000], seed=0, flags=oracle.NO_EFFICIENCY)
    _assert_records_equal({k2: v[:3000] for k2, v in a.items()}, ref, 3000)


def test_filter_first_and_in_flight_detect_the_same_fraction(toy):
    """PAPER.md:197 asks for this comparison.  On C2 (every photon's path is mirror -> detector) the two forms
    are draws of the same Bernoulli(R(lambda) QE(lambda)) per photon: detected counts agree within 4 sigma, at the full
    config size (1e7 photons), and the filter's kept count equals the sum of the oracle's probabilities likewise."""
    sc, gs = toy
    w = wl.make_config("C2")
    hm, ct = gs.alloc_accumulators()
    hm2, ct2 = gs.alloc_accumulators()
    step, kept, psum, pvar = 2_000_000, 0, 0.0, 0.0
    rec = gs.alloc_records(step)
    pre = None
    for a in range(0, w.n, step):
        o, d, lam = w.photon_range(a, a + step)
        do, dd, dl = _dev(o, d, lam)
        gs.propagate(do, dd, dl, seed=4, photon_id_base=a, records=rec, hitmap=hm, counters=ct)
        pre = gs.prefilter(do, dd, dl, [sc.info["m_mir"], sc.info["m_det"]], seed=4, photon_id_base=a, out=pre)
        gs.propagate(pre["origins"], pre["dirs"], pre["wavelengths"], seed=4, records=rec, hitmap=hm2, counters=ct2,
                     flags=opx.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"])
        kept += int(pre["n_kept"].item())
        if a == 0:                                                     # oracle probabilities on a sample of the ids
            p = oracle.prefilter(sc, lam[:200_000], [sc.info["m_mir"], sc.info["m_det"]], seed=4).prob.astype(np.float64)
            psum, pvar = p.sum(), (p * (1 - p)).sum()
            sample_keep = oracle.prefilter(sc, lam[:200_000], [sc.info["m_mir"], sc.info["m_det"]], seed=4).keep.sum()
            assert int((pre["index"][:int(pre["n_kept"].item())] < 200_000).sum().item()) == int(sample_keep)
            assert abs(sample_keep - psum) < 4 * np.sqrt(pvar)
    torch.cuda.synchronize()
    ct, ct2 = ct.cpu().numpy(), ct2.cpu().numpy()
    assert int(ct2[:7].sum()) == kept and int(ct[:7].sum()) == w.n
    n_flight, n_filter = int(ct[0]), int(ct2[0])
    sig = np.sqrt(max(n_flight, n_filter))
    assert abs(n_flight - n_filter) < 4 * np.sqrt(2) * sig, (n_flight, n_filter)
    assert n_filter > 0.9 * kept                                       # a kept photon is lost only to the dead border
    assert int(hm2.sum().item()) == n_filter
    # both hit-maps light the same ring
    lit, lit2 = (hm > 0).cpu().numpy(), (hm2 > 0).cpu().numpy()
    assert (lit & lit2).sum() > 0.9 * min(lit.sum(), lit2.sum())


# ------------------------------------------------------------------------------------ error paths
def test_filter_error_paths(toy):
    sc, gs = toy
    lib = pkg.load_library()
    x3, x1 = torch.zeros((64, 3), device="cuda"), torch.full((64,), 400.0, device="cuda")
    m_abs = next(i for i, m in enumerate(sc.materials) if m["kind"] == 0)
    with pytest.raises(pkg.OpxError) as e:
        gs.prefilter(x3, x3, x1, [sc.info["m_det"]] * 9)
    assert e.value.status == opx.OPX_ERR_INVALID_ARG
    with pytest.raises(pkg.OpxError):
        gs.prefilter(x3, x3, x1, [len(sc.materials)])
    with pytest.raises(pkg.OpxError):
        gs.prefilter(x3, x3, x1, [m_abs])
    with pytest.raises(pkg.OpxError):                                  # out must not alias in
        gs.prefilter(x3, x3, x1, [], out=dict(origins=x3, dirs=x3.clone(), wavelengths=x1.clone(), index=None,
                                              n_kept=torch.zeros(1, dtype=torch.int64, device="cuda")))
    need = C.c_size_t()
    assert lib.opx_prefilter_workspace_bytes(1 << 32, C.byref(need)) == opx.OPX_ERR_INVALID_ARG
    assert lib.opx_prefilter_workspace_bytes(64, C.byref(need)) == opx.OPX_OK and need.value >= 8 + 4
    fresh = pkg.Scene(sc)
    with pytest.raises(pkg.OpxError) as e:
        fresh.prefilter(x3, x3, x1, [])
    assert e.value.status == opx.OPX_ERR_BAD_STATE
    with pytest.raises(pkg.OpxError) as e:
        gs.propagate(x3, x3, x1, flags=2)
    assert e.value.status == opx.OPX_ERR_INVALID_ARG
    out = _host(gs.propagate(x3, x3, x1, flags=opx.FLAG_NO_EFFICIENCY))  # the library still works
    assert np.all(out["state"] == 6)


def test_large_scene_filtered_stream_kernel_shape_equals_small_calls(lhcb):
    """On a large scene a NO_EFFICIENCY call of >= 204 800 photons runs the 256-thread kernel shape (1024-photon tiles), smaller calls the
    512-photon-tile shape (which test_filter_then_trace_matches_oracle_c4 pins to the oracle on this scene): the same
    400 000 photons through one call and through two calls must give identical records, hit-maps and counters."""
    sc, gs = lhcb
    w = wl.make_config("C4")
    n = 400_000
    o, d, lam = w.photon_range(5_000_000, 5_000_000 + n)
    do, dd, dl = _dev(o, d, lam)
    one = _host(gs.propagate(do, dd, dl, flags=opx.FLAG_NO_EFFICIENCY))
    hm, ct = gs.alloc_accumulators()
    h = n // 2
    parts = [_host(gs.propagate(do[a:b].contiguous(), dd[a:b].contiguous(), dl[a:b].contiguous(), flags=opx.FLAG_NO_EFFICIENCY,
                                hitmap=hm, counters=ct)) for a, b in ((0, h), (h, n))]
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), one[k]), k
    assert np.array_equal(parts[-1]["hitmap"], one["hitmap"]) and np.array_equal(parts[-1]["counters"], one["counters"])
    assert int(one["counters"][:7].sum()) == n and not np.isin(one["state"], [1, 3]).any()
    # the same in flight: one call takes the 512-thread shape with 2048-photon tiles, the halves the small-call shape
    one_f = _host(gs.propagate(do, dd, dl, seed=3, photon_id_base=5_000_000))
    hm, ct = gs.alloc_accumulators()
    parts = [_host(gs.propagate(do[a:b].contiguous(), dd[a:b].contiguous(), dl[a:b].contiguous(), seed=3,
                                photon_id_base=5_000_000 + a, hitmap=hm, counters=ct)) for a, b in ((0, h), (h, n))]
    for k in ("state", "pixel", "surface", "bounces", "pos", "dir"):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), one_f[k]), k
    assert np.array_equal(parts[-1]["hitmap"], one_f["hitmap"]) and np.array_equal(parts[-1]["counters"], one_f["counters"])
    # and against the oracle on a sample of the one-call results
    idx = np.arange(0, n, 400)
    ref_f = oracle.trace_mesh(sc, o[idx], d[idx], lam[idx], seed=3, ids=(5_000_000 + idx).astype(np.uint64))
    for k in REC:
        assert np.array_equal(one_f[k][idx], ref_f[k]), k
    ref = oracle.trace_mesh(sc, o[idx], d[idx], lam[idx], flags=oracle.NO_EFFICIENCY)
    for k in REC:
        assert np.array_equal(one[k][idx], ref[k]), k
    assert np.array_equal(one["pos"][idx].astype(np.float64), ref["pos"])
