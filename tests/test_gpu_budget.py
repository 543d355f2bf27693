"""The 1e-5 mismatch budget on the large scene (north_star: "at most 1e-5 of photons may differ"; PAPER.md:173 is the
paper's own complaint about hit accuracy).  Zero mismatches among N photons bound the mismatch rate below 3/N at 95 %
confidence, so the budget needs N >= 3e5 photons compared against an all-triangle reference ON the 1.01e6-triangle scene
-- the scene with the deepest hierarchy, the most overlapping boxes (backing plates 1 mm behind every mirror facet) and
the one on which every culling shortcut of the traversal (padding, slack, beam widening, approximate reciprocals) works
hardest.

Per workload (C4: the 1e8 track photons of the headline; C5: the 1e9 mixed tracks):
  * 150 runs of 2048 CONSECUTIVE photon ids, the runs spread evenly over the whole id range: packets as coherent as in
    the bench launch (beam traversal of the 32-wide tree), both detector planes, every track of the source;
  * 100 000 single ids at a constant stride over the whole range: packets of unrelated rays (per-lane walk);
  -> 407 200 photons, product walk == GPU all-triangle loop (same arithmetic, no hierarchy) bit for bit on every record;
  * and the CPU oracle on every 20th of them (20 360 photons on C4, 10 180 on C5): bit-identical.
Together with tests/test_gpu_parity.py and test_gpu_robust.py that is > 1.1e6 photons on this scene with zero
mismatches allowed (95 % bound 2.7e-6)."""
import numpy as np
import pytest

import oracle
import paper_2309_12496_b200 as pkg
import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KEYS_INT = ("state", "surface", "pixel", "bounces")
RUNS, RUN_LEN, SINGLES = 150, 2048, 100_000


@pytest.fixture(scope="module")
def lhcb():
    sc = wl.lhcb_like_scene()
    return sc, pkg.Scene(sc).build()


def _sample_ids(n_total):
    starts = (np.arange(RUNS, dtype=np.uint64) * np.uint64((n_total - RUN_LEN) // (RUNS - 1)))
    runs = (starts[:, None] + np.arange(RUN_LEN, dtype=np.uint64)[None, :]).ravel()
    singles = np.uint64(17) + np.arange(SINGLES, dtype=np.uint64) * np.uint64((n_total - 17) // SINGLES)
    return np.concatenate([runs, singles])


def _host(out):
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


@pytest.mark.parametrize("config,oracle_every", [("C4", 20), ("C5", 40)])
def test_product_walk_equals_all_triangle_loop_on_4e5_photons_of_the_large_scene(lhcb, config, oracle_every):
    sc, gs = lhcb
    w = wl.make_config(config)
    assert w.scene.n_triangles == sc.n_triangles
    ids = _sample_ids(w.n)
    assert len(ids) == RUNS * RUN_LEN + SINGLES >= 400_000 and int(ids.max()) < w.n
    o, d, lam = w.photons(ids)
    do, dd, dl = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (o, d, lam))
    # the calls use id_base = 0: the random stream of entry i is keyed by i on all three sides
    prod = _host(gs.propagate(do, dd, dl, seed=13))
    assert pkg.last_kernel() == "k_propagate_packet<512, 4, 2, 0>"            # the shape the headline launch takes
    brute = _host(gs.propagate(do, dd, dl, seed=13, brute=True))
    mismatches = np.zeros(len(ids), bool)
    for k in KEYS_INT:
        mismatches |= prod[k] != brute[k]
    for k in ("pos", "dir"):
        x, y = prod[k].view(np.uint32), brute[k].view(np.uint32)
        mismatches |= (x != y).any(axis=1)
    assert mismatches.sum() == 0, f"{config}: {int(mismatches.sum())} of {len(ids)} photons differ, first at {np.flatnonzero(mismatches)[:5]}"
    assert np.array_equal(prod["hitmap"], brute["hitmap"]) and np.array_equal(prod["counters"][:7], brute["counters"][:7])
    # what the sample covers: every terminal state the scene produces, both mirror bounces, both detector planes
    assert len(np.unique(prod["state"])) >= 5 and prod["bounces"].max() == 2
    det = prod["pixel"][prod["state"] <= 1]
    assert det.min() < 32_000 <= det.max()
    # the oracle on a subset (state the subset): every `oracle_every`-th entry of the sample
    sub = np.arange(0, len(ids), oracle_every)
    ref = oracle.trace_mesh(sc, o[sub], d[sub], lam[sub], seed=13, ids=sub.astype(np.uint64))
    for k in KEYS_INT:
        assert np.array_equal(prod[k][sub], ref[k]), k
    assert np.array_equal(prod["pos"][sub].astype(np.float64), ref["pos"])
    assert np.array_equal(prod["dir"][sub].astype(np.float64), ref["dir"], equal_nan=True)
