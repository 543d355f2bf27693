"""Pins of the oracle's SURVEY.md 8(f) rows f1 (pre-propagation efficiency filter) and
f2 (histogram tables) against things other than the oracle: NumPy bin look-ups, closed-form
acceptance probabilities, binomial counts, and the paper's own justification of the filter ("any discarded
photons would not be detected"): filtering first and tracing without efficiencies detects the same fraction
as drawing in flight.  CPU only.  P-numbers continue DESIGN.md section 6.
"""
import numpy as np
import pytest

import oracle
import workloads as wl
from workloads.scenes import TABLE_HISTOGRAM, paper_histogram_tables, toy_rich_scene


# --------------------------------------------------------------------------- P15 histogram tables
def test_p15_histogram_bins_against_numpy():
    rng = np.random.default_rng(5)
    y = rng.random(16).astype(np.float32)                      # 16 bins of 25 nm over 200-600
    edges = 200.0 + 25.0 * np.arange(17)
    lam = np.concatenate([rng.uniform(200, 600, 2000), edges[:-1], edges[:-1] + 12.5]).astype(np.float32)
    want = y[np.clip(np.searchsorted(edges, lam.astype(np.float64), side="right") - 1, 0, 15)]
    for fp64 in (False, True):
        got = np.array([oracle.table_value(y, l, TABLE_HISTOGRAM, fp64=fp64) for l in lam], dtype=np.float32)
        assert np.array_equal(got, want)


def test_p15_histogram_edges_and_clamp():
    y = np.arange(16, dtype=np.float32) / 16
    tv = lambda l: oracle.table_value(y, l, TABLE_HISTOGRAM)
    assert tv(224.99) == y[0] and tv(225.0) == y[1]            # lower edge inclusive
    assert tv(200.0) == y[0] and tv(599.99) == y[15]
    assert tv(600.0) == y[15] and tv(1000.0) == y[15] and tv(100.0) == y[0]     # end bins extend outwards
    assert tv(float("nan")) == y[0]
    assert oracle.table_value(np.full(16, 0.37, np.float32), 431.0, TABLE_HISTOGRAM) == np.float32(0.37)


def test_p15_one_nm_grid_holds_the_papers_33_and_25_nm_binnings():
    refl, qe = paper_histogram_tables()
    assert refl.shape == qe.shape == (400,)
    # constant inside every 25 nm (33 nm) bin, stepping exactly at whole multiples of the bin width
    assert all(len(set(refl[k * 25:(k + 1) * 25])) == 1 for k in range(16))
    assert all(len(set(qe[k * 33:min(400, (k + 1) * 33)])) == 1 for k in range(13))
    assert len(set(refl)) == 16 and len(set(qe)) == 13
    assert abs(refl[0] - 0.94) < 1e-12 and abs(refl[-1] - 0.89) < 1e-12
    assert abs(qe.max() - 0.35) < 2e-3 and qe[250] == qe.max()                      # peak 35 % in the bin holding 450 nm
    sc = toy_rich_scene("paper_hist", cells=2)
    r32 = sc.materials[sc.info["m_mir"]]["table"]
    for lam, k in ((224.5, 0), (225.5, 1), (449.5, 9), (450.5, 10)):
        assert oracle.table_value(r32, lam, TABLE_HISTOGRAM) == r32[25 * k]


# ----------------------------------------------------------------------- P16 the filter's stream
def test_p16_filter_draw_is_stream_one_of_philox():
    for seed, g in ((0, 0), (7, 123456789), (0x299f31d0a4093822, 0x85a308d3243f6a88)):
        w0 = int(oracle.philox4x32_10([g & 0xffffffff, g >> 32, 0, 1], [seed & 0xffffffff, seed >> 32])[0])
        assert oracle.uniform_stream(seed, g, 0, 1) == (w0 >> 8) * 2.0 ** -24
        assert oracle.uniform_stream(seed, g, 0, 0) == oracle.uniform(seed, g, 0)
        assert oracle.uniform_stream(seed, g, 0, 1) != oracle.uniform(seed, g, 0)


def test_p16_keep_is_u_less_than_product():
    sc = toy_rich_scene("c2", cells=2)
    mir, det = sc.info["m_mir"], sc.info["m_det"]
    lam = np.linspace(190, 610, 500).astype(np.float32)
    r = oracle.prefilter(sc, lam, [mir, det, mir], seed=3, id_base=1000)
    R = np.array([oracle.table_lerp(sc.materials[mir]["table"], l) for l in lam], dtype=np.float32)
    Q = np.array([oracle.table_lerp(sc.materials[det]["table"], l) for l in lam], dtype=np.float32)
    p = (R * Q) * R                                             # left to right, each product rounded to fp32
    assert np.array_equal(r.prob, p)
    u = np.array([oracle.uniform_stream(3, 1000 + i, 0, 1) for i in range(len(lam))], dtype=np.float32)
    assert np.array_equal(r.keep, (u < p).astype(np.uint8))
    assert np.array_equal(r.index, np.flatnonzero(r.keep).astype(np.uint32))     # stable compaction


# ------------------------------------------------------------------- P17 acceptance probabilities
def test_p17_constant_tables_binomial_and_limits():
    sc = toy_rich_scene("flat", cells=2)
    mir, det = sc.info["m_mir"], sc.info["m_det"]
    n = 400_000
    lam = np.full(n, 333.0, np.float32)
    r = oracle.prefilter(sc, lam, [mir, det], seed=11)
    p = float(np.float32(0.9) * np.float32(0.25))
    assert r.prob[0] == np.float32(p)
    assert abs(len(r.index) - n * p) < 4 * np.sqrt(n * p * (1 - p))
    one, zero = toy_rich_scene("flat", cells=2), toy_rich_scene("flat", cells=2)
    for m in one.materials:
        m["table"] = np.ones_like(m["table"])
    for m in zero.materials:
        m["table"] = np.zeros_like(m["table"])
    assert len(oracle.prefilter(one, lam[:5000], [mir, det]).index) == 5000      # u < 1 always
    assert len(oracle.prefilter(zero, lam[:5000], [mir, det]).index) == 0        # u < 0 never
    assert len(oracle.prefilter(sc, lam[:5000], []).index) == 5000               # no factor: p = 1


def test_p17_wavelength_dependent_acceptance_matches_quadrature():
    sc = toy_rich_scene("c2", cells=2)
    mir, det = sc.info["m_mir"], sc.info["m_det"]
    n = 300_000
    lam = (200.0 + 400.0 * (np.arange(n) + 0.5) / n).astype(np.float32)          # uniform in wavelength
    kept = len(oracle.prefilter(sc, lam, [mir, det], seed=2).index)
    grid = np.linspace(200, 600, 64)
    fine = np.linspace(200, 600, 400001)
    R = np.interp(fine, grid, sc.materials[mir]["table"].astype(np.float64))
    Q = np.interp(fine, grid, sc.materials[det]["table"].astype(np.float64))
    p = np.trapezoid(R * Q, fine) / 400.0                                          # about 0.148
    assert 0.14 < p < 0.16
    assert abs(kept - n * p) < 4 * np.sqrt(n * p * (1 - p))


def test_p17_chunking_and_order_do_not_matter():
    sc = toy_rich_scene("c2", cells=2)
    f = [sc.info["m_mir"], sc.info["m_det"]]
    lam = np.random.default_rng(0).uniform(200, 600, 3000).astype(np.float32)
    whole = oracle.prefilter(sc, lam, f, seed=9, id_base=50)
    a, b = oracle.prefilter(sc, lam[:1234], f, seed=9, id_base=50), oracle.prefilter(sc, lam[1234:], f, seed=9, id_base=1284)
    assert np.array_equal(whole.keep, np.concatenate([a.keep, b.keep]))
    assert np.array_equal(whole.index, np.concatenate([a.index, b.index + 1234]))


# ------------------------------------------------- P18 filter first == draw in flight
def test_p18_filter_then_trace_detects_what_in_flight_detects():
    w = wl.make_config("C1", n=60_000)
    sc = w.scene
    o, d, lam = w.photon_range(0, w.n)
    flight = oracle.trace_mesh(sc, o, d, lam, seed=4)
    f = oracle.prefilter(sc, lam, [sc.info["m_mir"], sc.info["m_det"]], seed=4)
    k = f.index
    geo = oracle.trace_mesh(sc, o[k], d[k], lam[k], seed=4, ids=k.astype(np.uint64), flags=oracle.NO_EFFICIENCY)
    # every C1 photon's path is mirror -> detector pixel, so without efficiencies every traced photon is detected
    assert (geo.state == oracle.DETECTED).all() and (geo.bounces == 1).all()
    n, p = w.n, 0.225
    sig = np.sqrt(n * p * (1 - p))
    n_flight, n_filter = int(flight.counters[oracle.DETECTED]), int(geo.counters[oracle.DETECTED])
    assert abs(n_flight - n * p) < 4 * sig and abs(n_filter - n * p) < 4 * sig
    assert abs(n_flight - n_filter) < 4 * np.sqrt(2) * sig
    # geometry does not depend on the draws: where both forms detect a photon the records coincide
    both = np.flatnonzero(flight.state[k] == oracle.DETECTED)
    assert len(both) > 0.15 * len(k)
    for key in ("pos", "dir", "pixel", "surface"):
        assert np.array_equal(geo[key][both], flight[key][k[both]])
    # the two hit-maps are draws of the same distribution: compare the ring's radial profile
    assert abs(int(geo.hitmap.sum()) - n_filter) == 0
    assert set(np.flatnonzero(geo.hitmap)) <= set(np.flatnonzero(oracle.trace_mesh(sc, o, d, lam, seed=4, flags=oracle.NO_EFFICIENCY).hitmap))


def test_p18_no_efficiency_ignores_seed_and_never_rejects():
    w = wl.make_config("C3", n=40_000)
    ids = np.arange(0, w.n, 20, dtype=np.uint64)
    o, d, lam = w.photons(ids)
    a = oracle.trace_mesh(w.scene, o, d, lam, seed=1, ids=ids, flags=oracle.NO_EFFICIENCY)
    b = oracle.trace_mesh(w.scene, o, d, lam, seed=99, ids=ids + np.uint64(7), flags=oracle.NO_EFFICIENCY)
    for key in ("pos", "dir", "pixel", "surface", "state", "bounces"):
        assert np.array_equal(a[key], b[key])
    assert not np.isin(a.state, [oracle.QE_REJECTED, oracle.ABSORBED_MIRROR]).any()
    assert int(a.counters[:7].sum()) == len(ids)
    # an in-flight photon that was detected followed the same path
    c = oracle.trace_mesh(w.scene, o, d, lam, seed=1, ids=ids)
    det = c.state == oracle.DETECTED
    assert det.sum() > 50 and np.array_equal(a.pixel[det], c.pixel[det]) and (a.state[det] == oracle.DETECTED).all()


def test_histogram_scene_traces_with_bin_values():
    sc = toy_rich_scene("paper_hist", cells=6)
    w = wl.make_config("C1", n=4000)
    o, d, lam = w.photon_range(0, 4000)
    r = oracle.trace_mesh(sc, o, d, lam, seed=5)
    # replay the two draws of every photon with a NumPy bin look-up
    refl, qe = sc.materials[sc.info["m_mir"]]["table"], sc.materials[sc.info["m_det"]]["table"]
    j = np.clip(np.floor((lam.astype(np.float64) - 200.0)).astype(int), 0, 399)
    u0 = np.array([oracle.uniform(5, g, 0) for g in range(4000)], dtype=np.float32)
    u1 = np.array([oracle.uniform(5, g, 1) for g in range(4000)], dtype=np.float32)
    hit_mirror = r.bounces >= 1
    reached = (r.surface == 0) | hit_mirror
    want_absorbed = reached & ~(u0 < refl[j])
    assert np.array_equal(r.state == oracle.ABSORBED_MIRROR, want_absorbed)
    on_pixel = hit_mirror & (r.pixel >= 0)
    assert np.array_equal((r.state == oracle.DETECTED)[on_pixel], (u1 < qe[j])[on_pixel])
