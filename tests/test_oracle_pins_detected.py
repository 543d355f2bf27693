"""Pins of oracle.detected_list (the list of PAPER.md:195: "writes the position of the ray in a list when it interacts
with the detector").  The list is a filter of the tracer's records, so it is pinned against what the tracer computes
independently of its records -- the hit-map and the counters it accumulates inside its own loop (P4) -- against the
closed forms of the analytic toy RICH (P3, P6: ring radius, binomial detected count), and against invariants of a list
in photon order."""
import numpy as np

import oracle
import workloads as wl


def _trace(name, n, seed=3, id_base=0):
    w = wl.make_config(name, n=n)
    o, d, lam = w.photon_range(0, n)
    return w, oracle.trace_mesh(w.scene, o, d, lam, seed=seed, id_base=id_base)


def test_list_length_and_pixels_equal_the_tracers_own_counters_and_hitmap():
    w, r = _trace("C3", 3000)
    det = oracle.detected_list(r)
    assert len(det.id) == int(r.counters[oracle.DETECTED]) > 0
    assert np.array_equal(np.bincount(det.pixel, minlength=w.scene.n_pixels).astype(np.uint32), r.hitmap)
    assert det.pixel.min() >= 0


def test_list_is_in_photon_order_and_complete():
    _, r = _trace("C3", 3000, id_base=2 ** 40 + 17)
    det = oracle.detected_list(r, id_base=2 ** 40 + 17)
    assert det.id.dtype == np.uint64
    assert np.all(np.diff(det.id.astype(np.int64)) > 0)                  # strictly increasing: stable, no duplicates
    local = (det.id - np.uint64(2 ** 40 + 17)).astype(np.int64)
    mask = np.zeros(3000, bool)
    mask[local] = True
    assert np.all(r.state[mask] == oracle.DETECTED) and not np.any(r.state[~mask] == oracle.DETECTED)
    # explicit ids (a strided subset) are carried through
    ids = np.arange(0, 6000, 2, dtype=np.uint64)
    assert np.array_equal(oracle.detected_list(r, ids=ids).id, ids[local])


def test_c1_list_lies_on_the_focal_ring_with_the_binomial_count():
    """C1 closed forms: every listed hit is on the detector plane at ring radius ~ (R/2) tan(theta_c) from the ring centre
    (P3: 63.44 mm mean, 61.21 .. 65.43 mm astigmatic, each hit moved by at most a facet circumradius, P5), and the list holds R x QE = 0.9 x 0.25 of the photons within 4 sigma (P6)."""
    n = 4000
    w = wl.make_config("C1", n=n)
    o, d, lam = w.photon_range(0, n)
    r = oracle.trace_mesh(w.scene, o, d, lam, seed=0)
    det = oracle.detected_list(r)
    p = 0.9 * 0.25
    assert abs(len(det.id) - n * p) < 4 * np.sqrt(n * p * (1 - p))
    g = w.scene.info
    q = det.pos - g["D"]
    assert np.abs(q @ g["r"]).max() < 1e-2                               # on the detector plane
    centre = q.mean(axis=0)
    rad = np.linalg.norm(q - centre, axis=1)
    # P3: astigmatic ring radii 61.21 .. 65.43 mm about its centre; P5: a facet moves a hit by at most its circumradius 5.657 mm
    assert abs(rad.mean() - 0.5 * g["R"] * np.tan(0.0528842)) < 1.0
    assert rad.min() > 61.21 - 5.657 - 0.3 and rad.max() < 65.43 + 5.657 + 0.3
    # the arrival direction is the reflected chief ray within the cone angle
    assert np.all(np.arccos(np.clip(det.dir @ g["r"], -1, 1)) < 0.12)


def test_empty_and_no_efficiency():
    w, r = _trace("C3", 200)
    none = oracle.detected_list(dict(state=np.full(5, oracle.ESCAPED, np.uint8), pixel=np.full(5, -1, np.int32),
                                     pos=np.zeros((5, 3)), dir=np.zeros((5, 3))))
    assert len(none.id) == 0 and none.pos.shape == (0, 3)
    o, d, lam = w.photon_range(0, 200)
    r2 = oracle.trace_mesh(w.scene, o, d, lam, flags=oracle.NO_EFFICIENCY)
    det2 = oracle.detected_list(r2)
    # with efficiencies off every photon that reaches a pixel is listed: a superset of the in-flight list
    assert set(oracle.detected_list(r).id.tolist()) <= set(det2.id.tolist())
    assert len(det2.id) == int(r2.counters[oracle.DETECTED])
