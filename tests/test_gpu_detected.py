"""GPU parity of the detected-only output (opx_propagate_detected, opx_propagate_host_detected) against
oracle.detected_list on the same seeded inputs, through the C ABI.  Ids, pixels, positions and directions are copies of the
per-photon results, so the bar is bit-exact; the order is the photon-id order whatever the schedule."""
import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


@pytest.fixture(scope="module")
def toy():
    w = wl.make_config("C3", n=600_000)
    return w, pkg.Scene(w.scene).build()


def _check_list(got, k, ref):
    assert k == len(ref.id)
    assert np.array_equal(got["id"][:k].cpu().numpy().view(np.uint64), ref.id)
    assert np.array_equal(got["pixel"][:k].cpu().numpy(), ref.pixel)
    assert np.array_equal(got["pos"][:k].cpu().numpy().astype(np.float64), ref.pos)
    assert np.array_equal(got["dir"][:k].cpu().numpy().astype(np.float64), ref.dir)


@pytest.mark.parametrize("n", [1, 31, 512, 2049, 75_776, 100_003])
def test_detected_list_equals_the_oracles(toy, n):
    """Sizes around the tile sizes (512-photon and 1792-photon tiles, ragged tails) and a multi-wave launch."""
    w, gs = toy
    base = 2 ** 33 + 5
    o, d, lam = w.photon_range(1000, 1000 + n)
    out = gs.propagate_detected(*_dev(o, d, lam), seed=11, photon_id_base=base)
    torch.cuda.synchronize()
    ref = oracle.trace_mesh(w.scene, o, d, lam, seed=11, id_base=base)
    det = oracle.detected_list(ref, id_base=base)
    k = int(out["n_detected"].item())
    _check_list(out, k, det)
    assert np.array_equal(out["hitmap"].cpu().numpy().astype(np.uint32), ref.hitmap)
    assert np.array_equal(out["counters"].cpu().numpy().astype(np.uint64), ref.counters)


def test_calls_append_and_truncation_is_reported(toy):
    """Three chunked calls append to one list (= the list of one call); a list shorter than the detections holds `capacity`
    entries of the full list in increasing id, is untouched beyond, and still reports the true count."""
    w, gs = toy
    n = 60_000
    o, d, lam = w.photon_range(0, n)
    do, dd, dl = _dev(o, d, lam)
    one = gs.propagate_detected(do, dd, dl, seed=5)
    k = int(one["n_detected"].item())
    assert k > 100
    lst = gs.alloc_detected(n)
    hm, ct = gs.alloc_accumulators()
    for a, b in ((0, 7), (7, 41_000), (41_000, n)):
        gs.propagate_detected(do[a:b], dd[a:b], dl[a:b], seed=5, photon_id_base=a, out=lst, hitmap=hm, counters=ct)
    assert int(lst["n_detected"].item()) == k
    for key in ("id", "pixel", "pos", "dir"):
        assert torch.equal(lst[key][:k], one[key][:k]), key
    assert torch.equal(hm[:gs.n_pixels], one["hitmap"]) and torch.equal(ct, one["counters"])
    cap = k // 3
    small = gs.alloc_detected(cap + 8)
    for key in ("pixel",):
        small[key].fill_(-77)
    short = {key: (v[:cap] if key != "n_detected" else v) for key, v in small.items()}
    gs.propagate_detected(do, dd, dl, seed=5, out=short)
    assert int(short["n_detected"].item()) == k                       # true count, > capacity
    ids = short["id"].cpu().numpy()
    assert np.all(np.diff(ids) > 0)
    where = np.searchsorted(one["id"][:k].cpu().numpy(), ids)         # each kept entry is an entry of the full list
    for key in ("id", "pixel", "pos", "dir"):
        assert torch.equal(short[key].cpu(), one[key][:k].cpu()[where]), key
    assert bool((small["pixel"][cap:] == -77).all())                  # nothing written beyond the capacity


def test_detected_list_is_deterministic_and_matches_the_records(toy):
    """1e6 photons (multi-wave, every kernel shape's look-back chain is long): two runs give identical bytes, and the list is
    exactly the DETECTED subset of opx_propagate's records."""
    w, gs = toy
    n = 1_000_000
    steps = pkg.upload_track_steps(wl.make_config("C3", n=n).track_source.steps())
    o, d, lam = pkg.emit_cherenkov(steps, n, seed=2)
    a = gs.propagate_detected(o, d, lam, seed=9)
    b = gs.propagate_detected(o, d, lam, seed=9)
    rec = gs.propagate(o, d, lam, seed=9)
    torch.cuda.synchronize()
    k = int(a["n_detected"].item())
    assert k == int(b["n_detected"].item()) == int(rec["counters"][0].item())
    idx = torch.nonzero(rec["state"] == 0).flatten()
    assert torch.equal(a["id"][:k], idx)
    for key in ("pixel", "pos", "dir"):
        assert torch.equal(a[key][:k], b[key][:k]) and torch.equal(a[key][:k], rec[key][idx]), key
    assert torch.equal(a["hitmap"], rec["hitmap"])


def test_filtered_chain_and_device_side_count(toy):
    """emit + filter on the device, survivors traced with efficiencies off into a detected list (the count of survivors never
    leaves the device) == the oracle's chain."""
    w, gs = toy
    steps = w.track_source.steps()
    fac = [w.scene.info["m_det"], w.scene.info["m_mir"]]
    a, m = 40_000, 50_000
    pre = gs.emit_cherenkov_filtered(pkg.upload_track_steps(steps), m, fac, photon_id_base=a, seed=7)
    out = gs.propagate_detected(pre["origins"], pre["dirs"], pre["wavelengths"], flags=pkg.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"])
    # the same with the filter's index array: the list then names the ORIGINAL photons
    out2 = gs.propagate_detected(pre["origins"], pre["dirs"], pre["wavelengths"], flags=pkg.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"],
                                 index=pre["index"], photon_id_base=a)
    torch.cuda.synchronize()
    ro, rd, rl = oracle.emit_cherenkov(steps, m, id_base=a, seed=7)
    f = oracle.prefilter(w.scene, rl, fac, seed=7, id_base=a)
    ref = oracle.trace_mesh(w.scene, ro[f.index], rd[f.index], rl[f.index], flags=oracle.NO_EFFICIENCY)
    det = oracle.detected_list(ref)
    _check_list(out, int(out["n_detected"].item()), det)
    _check_list(out2, int(out2["n_detected"].item()), oracle.detected_list(ref, ids=np.uint64(a) + f.index.astype(np.uint64)))


@pytest.mark.parametrize("filtered", [False, True])
def test_from_track_steps_in_host_memory_to_the_detected_list(toy, filtered):
    """opx_tracks_host_detected (the loop memory-resident): step table in host memory in, detected list out,
    in chunks that split tiles and steps; == the oracle's chain emit (-> prefilter) -> trace -> detected_list, original ids."""
    w, gs = toy
    steps = w.track_source.steps()
    fac = [w.scene.info["m_det"], w.scene.info["m_mir"]] if filtered else []
    a, m = 123_456, 70_001
    got = gs.tracks_host_detected(steps, m, factors=fac, photon_id_base=a, seed=13, chunk=20_000)
    ro, rd, rl = oracle.emit_cherenkov(steps, m, id_base=a, seed=13)
    if filtered:
        f = oracle.prefilter(w.scene, rl, fac, seed=13, id_base=a)
        ref = oracle.trace_mesh(w.scene, ro[f.index], rd[f.index], rl[f.index], flags=oracle.NO_EFFICIENCY)
        det = oracle.detected_list(ref, ids=np.uint64(a) + f.index.astype(np.uint64))
    else:
        ref = oracle.trace_mesh(w.scene, ro, rd, rl, seed=13, id_base=a)
        det = oracle.detected_list(ref, id_base=a)
    k = got["n_detected"]
    assert k == len(det.id) > 50
    assert np.array_equal(got["id"][:k].numpy().view(np.uint64), det.id)
    assert np.array_equal(got["pixel"][:k].numpy(), det.pixel)
    assert np.array_equal(got["pos"][:k].numpy().astype(np.float64), det.pos)
    assert np.array_equal(got["dir"][:k].numpy().astype(np.float64), det.dir)
    assert np.array_equal(got["hitmap"][:gs.n_pixels].numpy().astype(np.uint32), ref.hitmap)
    assert np.array_equal(got["counters"].numpy().astype(np.uint64), ref.counters)


def test_host_path_detected(toy):
    """opx_propagate_host_detected: host buffers in, only the list + hit-map + counters out; chunked (ramped) uploads."""
    w, gs = toy
    n = 300_000
    o, d, lam = w.photon_range(0, n)
    dev = gs.propagate_detected(*_dev(o, d, lam), seed=4, photon_id_base=77)
    torch.cuda.synchronize()
    k = int(dev["n_detected"].item())
    pin = [torch.from_numpy(x).pin_memory() for x in (o, d, lam)]
    host = gs.propagate_host_detected(*pin, seed=4, photon_id_base=77, chunk=1 << 16)
    assert host["n_detected"] == k
    for key in ("id", "pixel", "pos", "dir"):
        assert torch.equal(host[key][:k], dev[key][:k].cpu()), key
    assert torch.equal(host["hitmap"][:gs.n_pixels], dev["hitmap"].cpu()) and torch.equal(host["counters"], dev["counters"].cpu())
    short = pkg.alloc_host_detected(k // 2, gs.n_pixels)
    res = gs.propagate_host_detected(*pin, seed=4, photon_id_base=77, chunk=1 << 16, out=short)
    kept = res["id"].numpy()
    assert res["n_detected"] == k and np.all(np.diff(kept) > 0) and np.isin(kept, dev["id"][:k].cpu().numpy()).all()


def test_detected_errors(toy):
    w, gs = toy
    o, d, lam = _dev(*w.photon_range(0, 64))
    lib = pkg.load_library()
    lst = gs.alloc_detected(64)
    with pytest.raises(pkg.OpxError):
        gs.propagate_detected(o, d, lam, flags=8)
    import ctypes as C
    from paper_2309_12496_b200 import opx
    dd = opx.Detected(*(lst[k].data_ptr() for k in ("id", "pixel", "pos", "dir")))
    hm, ct = gs.alloc_accumulators()
    ws = torch.empty(1 << 16, dtype=torch.uint8, device="cuda")
    args = lambda cap, nd, wsb: (gs._h, 64, None, 0, o.data_ptr(), d.data_ptr(), lam.data_ptr(), 0, 0, None, C.byref(dd), cap, nd,
                                 opx._aligned(ws), wsb, hm.data_ptr(), ct.data_ptr(), None)
    assert lib.opx_propagate_detected(*args(64, None, 1 << 15)) == opx.OPX_ERR_INVALID_ARG          # no length word
    assert lib.opx_propagate_detected(*args(0, lst["n_detected"].data_ptr(), 1 << 15)) == opx.OPX_ERR_INVALID_ARG   # capacity 0
    assert lib.opx_propagate_detected(*args(64, lst["n_detected"].data_ptr(), 0)) == opx.OPX_ERR_WORKSPACE_TOO_SMALL
    assert lib.opx_propagate_detected(*args(64, lst["n_detected"].data_ptr(), 1 << 15)) == opx.OPX_OK
