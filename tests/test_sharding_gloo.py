"""World-size-2 gloo test of the multi-GPU host logic (no GPU needed): contiguous id shards +
one sum all-reduce of hit-map and counters reproduce the single-rank result exactly.  The per-shard
records come from the oracle here (the CUDA path cannot run on CPU); what is under test is
paper_2309_12496_b200.sharding and the keying of the random stream by the global photon id."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import workloads as wl
from paper_2309_12496_b200.sharding import allreduce_accumulators, shard_range


def test_shard_range_tiles_exactly():
    for n, world in [(10, 3), (7, 8), (10_000_000, 8), (0, 2), (5, 1)]:
        spans = [shard_range(n, r, world) for r in range(world)]
        assert spans[0][0] == 0 and sum(c for _, c in spans) == n
        for (s0, c0), (s1, _) in zip(spans, spans[1:]):
            assert s0 + c0 == s1
        counts = [c for _, c in spans]
        assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _worker(rank, world, port, n_total, seed, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.make_config("C3", n=600_000)
    start, count = shard_range(n_total, rank, world)
    o, d, lam = w.photon_range(300_000 + start, 300_000 + start + count)
    r = oracle.trace_mesh(w.scene, o, d, lam, seed=seed, id_base=300_000 + start, n_threads=2)
    hitmap = torch.from_numpy(r["hitmap"].astype(np.int32))
    counters = torch.from_numpy(r["counters"].astype(np.int64))
    allreduce_accumulators(hitmap, counters)
    np.save(os.path.join(out_dir, f"state_{rank}.npy"), r["state"])
    det = oracle.detected_list(r, id_base=300_000 + start)               # the rank's shard of the detected list
    np.save(os.path.join(out_dir, f"det_id_{rank}.npy"), det.id)
    np.save(os.path.join(out_dir, f"det_pos_{rank}.npy"), det.pos)
    if rank == 0:
        np.save(os.path.join(out_dir, "hitmap.npy"), hitmap.numpy())
        np.save(os.path.join(out_dir, "counters.npy"), counters.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_reproduce_single_rank(tmp_path):
    n_total, seed, world = 3001, 13, 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(world, port, n_total, seed, str(tmp_path)), nprocs=world, join=True)
    w = wl.make_config("C3", n=600_000)
    o, d, lam = w.photon_range(300_000, 300_000 + n_total)
    ref = oracle.trace_mesh(w.scene, o, d, lam, seed=seed, id_base=300_000)
    state = np.concatenate([np.load(tmp_path / f"state_{r}.npy") for r in range(world)])
    assert np.array_equal(state, ref["state"])
    assert np.array_equal(np.load(tmp_path / "hitmap.npy").astype(np.uint32), ref["hitmap"])
    assert np.array_equal(np.load(tmp_path / "counters.npy").astype(np.uint64), ref["counters"])
    assert ref["hitmap"].sum() > 0
    # the detected lists stay sharded: concatenated in rank order they are the single-rank list (ids increasing across ranks)
    det = oracle.detected_list(ref, id_base=300_000)
    assert np.array_equal(np.concatenate([np.load(tmp_path / f"det_id_{r}.npy") for r in range(world)]), det.id)
    assert np.array_equal(np.concatenate([np.load(tmp_path / f"det_pos_{r}.npy") for r in range(world)]), det.pos)


def _worker_chain(rank, world, port, n_total, seed, out_dir):
    """Rows F4 + F1 under sharding: each rank generates ITS id range from the replicated step table, filters it and
    traces the survivors; only the hit-map and the counters are exchanged."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.make_config("C3", n=200_000)
    steps = w.track_source.steps()
    start, count = shard_range(n_total, rank, world)
    o, d, lam = oracle.emit_cherenkov(steps, count, id_base=100_000 + start, seed=seed)
    f = oracle.prefilter(w.scene, lam, [w.scene.info["m_det"], w.scene.info["m_mir"]], seed=seed, id_base=100_000 + start)
    r = oracle.trace_mesh(w.scene, o[f.index], d[f.index], lam[f.index], flags=oracle.NO_EFFICIENCY, n_threads=2)
    hitmap = torch.from_numpy(r["hitmap"].astype(np.int32))
    counters = torch.from_numpy(r["counters"].astype(np.int64))
    allreduce_accumulators(hitmap, counters)
    np.save(os.path.join(out_dir, f"kept_{rank}.npy"), f.index.astype(np.int64) + start)
    if rank == 0:
        np.save(os.path.join(out_dir, "hitmap.npy"), hitmap.numpy())
        np.save(os.path.join(out_dir, "counters.npy"), counters.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_emit_filter_trace_chain_reproduces_single_rank(tmp_path):
    n_total, seed, world = 4001, 21, 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker_chain, args=(world, port, n_total, seed, str(tmp_path)), nprocs=world, join=True)
    w = wl.make_config("C3", n=200_000)
    o, d, lam = oracle.emit_cherenkov(w.track_source.steps(), n_total, id_base=100_000, seed=seed)
    f = oracle.prefilter(w.scene, lam, [w.scene.info["m_det"], w.scene.info["m_mir"]], seed=seed, id_base=100_000)
    ref = oracle.trace_mesh(w.scene, o[f.index], d[f.index], lam[f.index], flags=oracle.NO_EFFICIENCY)
    kept = np.concatenate([np.load(tmp_path / f"kept_{r}.npy") for r in range(world)])
    assert np.array_equal(kept, f.index.astype(np.int64))               # the same photons survive, in the same order
    assert np.array_equal(np.load(tmp_path / "hitmap.npy").astype(np.uint32), ref["hitmap"])
    assert np.array_equal(np.load(tmp_path / "counters.npy").astype(np.uint64), ref["counters"])
    assert ref["hitmap"].sum() > 100


def test_bench_id_ranges_for_two_and_eight_ranks():
    """bench.py's weak-scaling arithmetic without CUDA: rank r of `world` takes shard_range(n * world, r, world) of a job of
    n photons per GPU; the ranges are n photons each, contiguous, and tile ids [0, n * world) for world = 2 and 8 (the sizes
    the driver's scaling run uses) -- also when n is not a multiple of anything."""
    for world in (2, 8):
        for n in (100_000_000, 600_000, 12_345_677):
            spans = [shard_range(n * world, r, world) for r in range(world)]
            assert [c for _, c in spans] == [n] * world
            assert [s for s, _ in spans] == [r * n for r in range(world)]
