"""GPU parity for SURVEY.md 8(f) row f4: on-device Cherenkov generation from track steps through the
C ABI against oracle.emit_cherenkov on the same step tables.  IEEE operations only on both sides (no sin/cos), so the
bar is bit-exact on every output float; the generated arrays then feed opx_propagate / opx_prefilter without leaving
the device and the records are compared with the oracle's emit -> trace chain."""
import ctypes as C

import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl
from paper_2309_12496_b200 import opx

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _bits(t):
    return t.cpu().numpy().view(np.uint32)


def _assert_same_bits(got, ref):
    for g, r, name in zip(got, ref, ("origins", "dirs", "wavelengths")):
        assert np.array_equal(_bits(g), np.ascontiguousarray(r).view(np.uint32)), name


def _random_steps(rng, S, counts, beta=None):
    w = rng.normal(size=(S, 3))
    w[:6] = [[0, 0, 1], [0, 0, -1], [1, 0, 0], [0, -1, 0], [0.6, 0, -0.8], [1e-4, 1e-4, -1]]
    w /= np.linalg.norm(w, axis=1, keepdims=True)
    return dict(x=rng.uniform(-100, 100, (S, 3)).astype(np.float32), w=w.astype(np.float32),
                length=rng.uniform(0.1, 5.0, S).astype(np.float32),
                beta=(rng.uniform(0.9980, 1.0, S) if beta is None else np.asarray(beta)).astype(np.float32),
                first=np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64))


def test_emit_matches_oracle_bit_for_bit():
    """Random steps in both hemispheres and at the poles of the frame, beta above / at / below threshold, steps
    without photons, a 64-bit seed; ~1e5 photons, ragged against the 256-thread blocks."""
    rng = np.random.default_rng(41)
    S = 1500
    counts = rng.integers(0, 140, S)
    counts[[3, 4, 17, S - 1]] = 0
    counts[200:900] = 0                                # a block of photons that spans 700 steps without photons
    counts[950:1300:2] = 0
    beta = rng.uniform(0.9980, 1.0, S)
    beta[:8] = [1.0, 0.99860196, 0.9986, 0.5, 0.9, 1.0, 1.0, 1.0]
    st = _random_steps(rng, S, counts, beta)
    n, seed = int(st["first"][-1]), (0xFEEDBEEF << 32) | 0x1234567
    ref = oracle.emit_cherenkov(st, n, seed=seed)
    ds = pkg.upload_track_steps(st)
    got = pkg.emit_cherenkov(ds, n, seed=seed)
    _assert_same_bits(got, ref)
    # chunks and id bases: the same bits
    parts = [pkg.emit_cherenkov(ds, b - a, photon_id_base=a, seed=seed) for a, b in ((0, 1), (1, 257), (257, n))]
    for k in range(3):
        assert torch.equal(torch.cat([p[k] for p in parts]), got[k])
    assert not torch.equal(pkg.emit_cherenkov(ds, n, seed=seed + 1)[1], got[1])


def test_emit_c3_workload_sampled_parity_and_properties_at_full_size():
    """The C3 workload's own step table (1e7 photons, 3.4e5 steps): GPU == oracle on three id ranges incl. the very
    last photons; on all 1e7 photons the closed forms of P22/P24 hold (theta_c, unit length, spectrum range and mean,
    every photon on its own 1 mm step)."""
    w = wl.make_config("C3")
    st = w.track_source.steps()
    ds = pkg.upload_track_steps(st)
    assert ds["n_total"] == w.n
    for a, m in ((0, 50_000), (4_999_871, 30_000), (w.n - 20_011, 20_011)):
        _assert_same_bits(pkg.emit_cherenkov(ds, m, photon_id_base=a, seed=5), oracle.emit_cherenkov(st, m, id_base=a, seed=5))
    o, d, lam = pkg.emit_cherenkov(ds, w.n, seed=5)
    step = torch.searchsorted(ds["first"], torch.arange(w.n, device="cuda"), right=True) - 1
    wv = ds["w"][step].double()
    cosang = (d.double() * wv).sum(dim=1)
    assert float((cosang - 1 / 1.0014).abs().max()) < 3e-7
    assert float((d.double().norm(dim=1) - 1).abs().max()) < 2.0 ** -22
    assert float(lam.min()) >= 200.0 and float(lam.max()) <= 600.0 and abs(float(lam.double().mean()) - 329.58) < 0.1
    rel = o.double() - ds["x"][step].double()
    frac = (rel * wv).sum(dim=1)
    assert float(frac.min()) > -1e-4 and float(frac.max()) < 1 + 1e-4 and abs(float(frac.mean()) - 0.5) < 1e-3
    assert float((rel - frac[:, None] * wv).abs().max()) < 1e-4


def test_emit_then_propagate_matches_the_oracle_chain():
    """Generation and propagation chained on the device (no host copy of a photon) against oracle.emit_cherenkov ->
    oracle.trace_mesh, and likewise through the paper's filter: identical records, hit-map and counters."""
    w = wl.make_config("C3", n=2_000_000)
    st = w.track_source.steps()
    ds = pkg.upload_track_steps(st)
    gs = pkg.Scene(w.scene).build()
    a, m = 1_234_567, 20_000
    o, d, lam = pkg.emit_cherenkov(ds, m, photon_id_base=a, seed=8)
    got = gs.propagate(o, d, lam, seed=8, photon_id_base=a)
    ro, rd, rl = oracle.emit_cherenkov(st, m, id_base=a, seed=8)
    ref = oracle.trace_mesh(w.scene, ro, rd, rl, seed=8, id_base=a)
    torch.cuda.synchronize()
    for k in ("state", "surface", "pixel", "bounces"):
        assert np.array_equal(got[k].cpu().numpy(), ref[k]), k
    assert np.array_equal(got["pos"].cpu().numpy().astype(np.float64), ref["pos"])
    assert np.array_equal(got["hitmap"].cpu().numpy(), ref["hitmap"])
    assert np.array_equal(got["counters"].cpu().numpy().astype(np.uint64), ref["counters"])
    assert len(np.unique(ref["state"])) >= 3                      # one track: detected, QE-rejected, mirror-absorbed
    fac = [w.scene.info["m_det"], w.scene.info["m_mir"]]
    pre = gs.prefilter(o, d, lam, fac, seed=8, photon_id_base=a)
    geo = gs.propagate(pre["origins"], pre["dirs"], pre["wavelengths"], flags=opx.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"])
    f = oracle.prefilter(w.scene, rl, fac, seed=8, id_base=a)
    rgeo = oracle.trace_mesh(w.scene, ro[f.index], rd[f.index], rl[f.index], flags=oracle.NO_EFFICIENCY)
    k = len(f.index)
    assert int(pre["n_kept"].item()) == k
    for key in ("state", "surface", "pixel", "bounces"):
        assert np.array_equal(geo[key][:k].cpu().numpy(), rgeo[key]), key
    assert np.array_equal(geo["hitmap"].cpu().numpy(), rgeo["hitmap"])


def test_emit_error_paths():
    rng = np.random.default_rng(2)
    st = _random_steps(rng, 10, [5] * 10)
    ds = pkg.upload_track_steps(st)
    for kwargs in (dict(n=51), dict(n=1, photon_id_base=50), dict(n=5, lambda1=0.0), dict(n=5, lambda1=600.0, lambda2=200.0),
                   dict(n=5, n_index=float("nan"))):
        with pytest.raises(pkg.OpxError) as e:
            pkg.emit_cherenkov(ds, **kwargs)
        assert e.value.status == opx.OPX_ERR_INVALID_ARG
    assert pkg.emit_cherenkov(ds, 0)[2].numel() == 0
    lib = pkg.load_library()
    assert lib.opx_emit_cherenkov(None, 50, 1.0014, 200.0, 600.0, 5, 0, 0, None, None, None, None) == opx.OPX_ERR_INVALID_ARG
    empty = opx.TrackSteps()
    x = torch.zeros(16, device="cuda")
    assert lib.opx_emit_cherenkov(C.byref(empty), 0, 1.0014, 200.0, 600.0, 1, 0, 0, C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()),
                                  C.c_void_p(x.data_ptr()), None) == opx.OPX_ERR_INVALID_ARG
    o, d, lam = pkg.emit_cherenkov(ds, 50, seed=1)                       # still works afterwards
    assert torch.isfinite(d).all()


def test_fused_emit_filter_equals_the_two_calls_and_the_oracle_chain():
    """opx_emit_cherenkov_filtered == opx_emit_cherenkov then opx_prefilter == oracle.emit_cherenkov then
    oracle.prefilter: survivor count, ids (stable order) and every bit of the survivors' photons; block boundaries
    (2048 ids), a ragged tail, a 64-bit id base into the table, K = 0 (everything kept) and n = 0."""
    w = wl.make_config("C3", n=3_000_000)
    st = w.track_source.steps()
    ds = pkg.upload_track_steps(st)
    gs = pkg.Scene(w.scene).build()
    fac = [w.scene.info["m_det"], w.scene.info["m_mir"], w.scene.info["m_mir"]]
    for a, m in ((0, 1), (5, 2048), (2_000_001, 2049), (1_111_111, 300_037)):
        fused = gs.emit_cherenkov_filtered(ds, m, fac, photon_id_base=a, seed=6)
        o, d, lam = pkg.emit_cherenkov(ds, m, photon_id_base=a, seed=6)
        two = gs.prefilter(o, d, lam, fac, seed=6, photon_id_base=a)
        k = int(fused["n_kept"].item())
        assert k == int(two["n_kept"].item())
        for key in ("origins", "dirs", "wavelengths", "index"):
            assert torch.equal(fused[key][:k], two[key][:k]), key
        ro, rd, rl = oracle.emit_cherenkov(st, m, id_base=a, seed=6)
        f = oracle.prefilter(w.scene, rl, fac, seed=6, id_base=a)
        assert k == len(f.index) and np.array_equal(fused["index"][:k].cpu().numpy().view(np.uint32), f.index)
        _assert_same_bits((fused["origins"][:k], fused["dirs"][:k], fused["wavelengths"][:k]), (ro[f.index], rd[f.index], rl[f.index]))
    allk = gs.emit_cherenkov_filtered(ds, 5000, [], photon_id_base=77, seed=6)
    assert int(allk["n_kept"].item()) == 5000
    _assert_same_bits((allk["origins"], allk["dirs"], allk["wavelengths"]), oracle.emit_cherenkov(st, 5000, id_base=77, seed=6))
    none = gs.emit_cherenkov_filtered(ds, 0, fac, out=dict(allk, n_kept=torch.full((1,), 9, dtype=torch.int64, device="cuda")))
    assert int(none["n_kept"].item()) == 0
    # the chain to hits: survivors traced with efficiencies off == the oracle's chain
    a, m = 1_500_000, 40_000
    fused = gs.emit_cherenkov_filtered(ds, m, fac[:2], photon_id_base=a, seed=2, capacity=m // 2)
    geo = gs.propagate(fused["origins"], fused["dirs"], fused["wavelengths"], flags=opx.FLAG_NO_EFFICIENCY, n_dev=fused["n_kept"])
    ro, rd, rl = oracle.emit_cherenkov(st, m, id_base=a, seed=2)
    f = oracle.prefilter(w.scene, rl, fac[:2], seed=2, id_base=a)
    ref = oracle.trace_mesh(w.scene, ro[f.index], rd[f.index], rl[f.index], flags=oracle.NO_EFFICIENCY)
    k = len(f.index)
    for key in ("state", "surface", "pixel", "bounces"):
        assert np.array_equal(geo[key][:k].cpu().numpy(), ref[key]), key
    assert np.array_equal(geo["hitmap"].cpu().numpy(), ref["hitmap"])
    with pytest.raises(pkg.OpxError):
        gs.emit_cherenkov_filtered(ds, 10, [len(w.scene.materials)])
    with pytest.raises(pkg.OpxError):
        gs.emit_cherenkov_filtered(ds, 10, fac, photon_id_base=ds["n_total"] - 5)
