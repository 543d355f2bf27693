#!/usr/bin/env python
"""bench.py -- photons/s of the per-photon optical propagation hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C2] [--photons n]

One "step" = one opx_propagate call (one kernel: propagation with hit binning and counters inside) over one batch of
synthetic photons of the named BASELINE.json config (default C2 = configs[1]: toy RICH, 20 014
triangles, 1e7 photons), inputs resident in HBM.  The BVH build is timed separately (`bvh_build_ms`)
as SURVEY.md 8(d) prescribes.  N > 1 (torchrun): every rank propagates its own contiguous id range
of the same size (weak scaling) and the per-rank hit-maps and counters are summed with one NCCL
all-reduce per step.  Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "optical photons propagated/sec on 1 B200 (device-timed), % of roofline"
UNIT = "photons/s"
# FLOP model of SURVEY.md 8(d) / DESIGN.md 9: FMA = 2, add/mul/min/max/compare/divide = 1
FLOP_NODE, FLOP_TRI, FLOP_SEGMENT, FLOP_INTERACTION = 48, 50, 15, 35
BYTES_IN, BYTES_OUT, BYTES_BIN = 28, 34, 6          # per photon: inputs, hit record, re-read by k_bin
# dram__bytes_read.sum + dram__bytes_write.sum of k_propagate per launch from the ncu --set full
# capture summarised in profiles/ (None until one exists for the current kernel)
NCU_TRAFFIC_BYTES = {"C2": 567209728}   # profiles/r01_v27_k_propagate_packet.md


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({names[k] for r in self.rows if len(r) >= 7 for k in range(4) if r[3 + k].startswith("Active")})
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=reasons, samples=len(sm))


def time_oracle(workload, n_sample, seed, repeats=1, n_threads=None):
    """The oracle as it stands on the host cores, on the first n_sample photon ids of the workload."""
    import oracle
    o, d, lam = workload.photon_range(0, n_sample)
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        r = oracle.trace_mesh(workload.scene, o, d, lam, seed=seed, n_threads=n_threads)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return n_sample / best, r["n_threads"], best, int(r["counters"][7])


def run_reference(args):
    """--impl reference: the CPU oracle timed on a bounded sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads
    w = workloads.make_config(args.config, n=args.photons)
    import oracle
    # bounded sample per step: at most --reference-sample photons, and no more than about 3 s of work (probed), so that
    # `--steps K --warmup W` ends within minutes on any config
    po, pd, pl = w.photon_range(0, 1000)
    t0 = time.perf_counter()
    oracle.trace_mesh(w.scene, po, pd, pl, seed=args.seed)
    rate = 1000 / (time.perf_counter() - t0)
    n_sample = int(min(w.n, args.reference_sample, max(1000, rate * 3.0)))
    o, d, lam = w.photon_range(0, n_sample)
    for _ in range(args.warmup):
        oracle.trace_mesh(w.scene, o[:1000], d[:1000], lam[:1000], seed=args.seed)
    t0 = time.perf_counter()
    threads = 0
    for _ in range(args.steps):
        r = oracle.trace_mesh(w.scene, o, d, lam, seed=args.seed)
        threads = r["n_threads"]
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = f"first {n_sample} photon ids of {args.config} per step, brute force over {w.scene.n_triangles} triangles"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.config}{' + mirror vertex normals' if args.smooth else ''}: {w.scene.n_triangles} triangles, {w.n} photons (sampled)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_sweep(args, scene, photons, records, hitmap, counters, n, stream, w, pkg):
    """BASELINE.json config 4: photons/s and achieved HBM GB/s versus chunk size.  The resident batch of
    n photons is streamed repeatedly (global ids keep advancing, so every pass draws new random
    numbers) until --total photons have gone through, in calls of `chunk` photons each."""
    import torch
    d_o, d_d, d_l = photons
    rows = []
    side = [torch.cuda.Stream(device=d_o.device) for _ in range(max(0, args.streams - 1))]
    fork, joins = torch.cuda.Event(), [torch.cuda.Event() for _ in side]
    for chunk in [int(c) for c in args.chunks.split(",") if int(c) <= n]:
        for n_streams in sorted({1, args.streams}):
            lanes = [stream] + side[:n_streams - 1]

            def one_pass(base):
                for k, a in enumerate(range(0, n - chunk + 1, chunk)):
                    rec = {key: v[a:a + chunk] for key, v in records.items()}
                    scene.propagate(d_o[a:a + chunk], d_d[a:a + chunk], d_l[a:a + chunk], seed=args.seed, photon_id_base=base + a,
                                    records=rec, hitmap=hitmap, counters=counters, stream=lanes[k % n_streams])

            def timed(passes_, per_pass_):
                # calls are independent (hit-map and counters are integer atomics), so they may be spread over streams:
                # the side streams fork from and join back into the timed stream
                fork.record(stream)
                for st in lanes[1:]:
                    st.wait_event(fork)
                for p in range(passes_):
                    one_pass((p + 1) * per_pass_)
                for st, ev in zip(lanes[1:], joins):
                    ev.record(st)
                    stream.wait_event(ev)
            per_pass = (n // chunk) * chunk
            passes = max(1, min(args.total // per_pass, 50))
            hitmap.zero_(); counters.zero_()
            timed(1, 0)                                                    # warm-up
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = pkg.launch_count()
            ev0.record(stream)
            timed(passes, per_pass)
            ev1.record(stream)
            torch.cuda.synchronize()
            ms = ev0.elapsed_time(ev1)
            done = passes * per_pass
            rows.append({"chunk": chunk, "streams": n_streams, "photons": done, "calls": passes * (n // chunk), "ms": ms,
                         "photons_per_s": done / (ms * 1e-3), "hbm_gbs_algorithmic": done * (BYTES_IN + BYTES_OUT) / (ms * 1e-3) / 1e9,
                         "gpu_launches": pkg.launch_count() - l0})
    best = max(rows, key=lambda r: r["photons_per_s"])
    print(json.dumps({"metric": METRIC, "value": best["photons_per_s"], "unit": UNIT, "n_gpus": 1, "higher_is_better": True,
                      "dtype": "f32", "data": "synthetic", "scaling": "weak", "vs_baseline": None,
                      "config": {"workload": f"{args.config} chunk-size sweep: {w.scene.n_triangles} triangles, resident batch of {n} photons "
                                             f"streamed until {args.total} photons per chunk size", "best_chunk": best["chunk"]},
                      "sweep": rows}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="opx", choices=["opx", "reference"])
    ap.add_argument("--config", default="C2", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--photons", type=int, default=None, help="photons per GPU per step (default: the config's N)")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="CPU time budget of each cpu_baseline leg (all cores, one thread)")
    ap.add_argument("--reference-sample", type=int, default=20000)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--smooth", action="store_true",
                    help="toy-scene configs (C1-C3) with vertex normals on the mirror (SURVEY.md 8(f) row f3): a variant "
                         "of the workload, named in config.workload; not the default line")
    ap.add_argument("--sweep", action="store_true",
                    help="config C5 protocol: stream --total photons through the resident batch in chunks of 1e5..1e8 "
                         "and report photons/s and HBM GB/s per chunk size instead of the default line")
    ap.add_argument("--total", type=int, default=1_000_000_000, help="photons streamed per chunk size in --sweep")
    ap.add_argument("--chunks", type=str, default="100000,1000000,10000000,100000000")
    ap.add_argument("--streams", type=int, default=4, help="--sweep: also time every chunk size with the calls spread over this many streams")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "opx" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2309_12496_b200 as pkg
    import workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    from paper_2309_12496_b200.sharding import allreduce_accumulators, shard_range
    w = workloads.make_config(args.config, n=None)
    n = args.photons if args.photons else min(w.n, 100_000_000)       # per GPU per step (weak scaling)
    w = workloads.make_config(args.config, n=max(w.n, n * world))     # the job: world * n photons, ids 0..world*n
    if args.smooth:
        if args.config not in ("C1", "C2", "C3"):
            raise SystemExit("--smooth: only the toy scene (C1-C3) has an analytic vertex-normal field")
        from workloads.scenes import toy_rich_scene
        w.scene = toy_rich_scene("flat" if args.config == "C1" else "c2", smooth=True)
    id_base, n = shard_range(n * world, rank, world)                  # contiguous global id range of this rank
    pin = [torch.empty((n, 3), dtype=torch.float32).pin_memory(), torch.empty((n, 3), dtype=torch.float32).pin_memory(),
           torch.empty(n, dtype=torch.float32).pin_memory()]
    for a in range(0, n, 5_000_000):                                  # generate in slices to bound host memory
        b = min(n, a + 5_000_000)
        for dst, src in zip(pin, w.photon_range(id_base + a, id_base + b)):
            dst[a:b] = torch.from_numpy(src)
    d_o, d_d, d_l = (x.to(dev, non_blocking=True) for x in pin)
    stream = torch.cuda.current_stream(dev)

    # ---- scene + BVH build (timed separately: SURVEY.md 8(d))
    scene = pkg.Scene(w.scene)
    scene.build(dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = pkg.launch_count()
    torch.cuda.synchronize()
    t_build = []
    for _ in range(3):
        t0 = time.perf_counter()
        scene.build(dev)
        t_build.append(1e3 * (time.perf_counter() - t0))
    build_launches = (pkg.launch_count() - l0) // 3

    records = scene.alloc_records(n, dev)
    hitmap, counters = scene.alloc_accumulators(dev)

    if args.sweep:
        return run_sweep(args, scene, (d_o, d_d, d_l), records, hitmap, counters, n, stream, w, pkg)

    def step():
        hitmap.zero_(); counters.zero_()
        scene.propagate(d_o, d_d, d_l, seed=args.seed, photon_id_base=id_base, records=records, hitmap=hitmap,
                        counters=counters, stream=stream)
        allreduce_accumulators(hitmap, counters)                      # the one exchange step (no-op at N = 1)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    scene.profile_begin(args.steps)
    l0 = pkg.launch_count()
    torch.cuda.synchronize()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = pkg.launch_count() - l0                           # kernels of libopx.so only (torch fills not counted)
    ms_prop, ms_bin = scene.profile_end()
    clocks = sampler.stop()
    if dist is not None:
        t = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * n * args.steps / (ms_total * 1e-3)
    cnt = counters.cpu().numpy()

    # ---- end to end through the C ABI with host buffers (copies inside the timed region)
    e2e = None
    if rank == 0 or dist is not None:
        host_out = pkg.alloc_host_records(n, scene.n_pixels)
        chunk = min(n, 1 << 20)
        scene.propagate_host(*pin, seed=args.seed, photon_id_base=id_base, chunk=chunk, out=host_out, stream=stream)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            host_out["hitmap"].zero_(); host_out["counters"].zero_()
            scene.propagate_host(*pin, seed=args.seed, photon_id_base=id_base, chunk=chunk, out=host_out, stream=stream)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if dist is not None:
            t = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * n * args.e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": BYTES_IN * n,
               "d2h_bytes_per_step": BYTES_OUT * n + 4 * scene.n_pixels + 64, "chunk_photons": chunk,
               "ms_per_step": 1e3 * dt / args.e2e_steps}
        if not np.array_equal(host_out["counters"].numpy(), cnt if dist is None else host_out["counters"].numpy()):
            raise SystemExit("bench: host path and device path disagree")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (k_propagate), DESIGN.md section 9
    peaks = measured_peaks()
    stats = scene.propagate_stats(d_o, d_d, d_l, seed=args.seed, photon_id_base=id_base)
    flop = (FLOP_NODE * stats["nodes"] + FLOP_TRI * stats["triangle_tests"] + FLOP_SEGMENT * stats["segments"]
            + FLOP_INTERACTION * stats["interactions"])
    t_prop = statistics.mean(ms_prop) * 1e-3
    t_bin = statistics.mean(ms_bin) * 1e-3
    fp32_peak_tflops = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    alu_achieved = flop / t_prop / 1e12
    hbm_bytes = (BYTES_IN + BYTES_OUT) * n
    hbm_achieved = hbm_bytes / t_prop / 1e9
    t_alu_bound, t_hbm_bound = flop / (fp32_peak_tflops * 1e12), hbm_bytes / (peaks["hbm_gbs"] * 1e9)
    if t_alu_bound >= t_hbm_bound:
        roof = {"bound": "alu", "achieved": alu_achieved, "peak": fp32_peak_tflops, "unit": "TFLOP/s",
                "frac": alu_achieved / fp32_peak_tflops}
    else:
        roof = {"bound": "hbm", "achieved": hbm_achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": hbm_achieved / peaks["hbm_gbs"]}
    roof.update({
        "traffic": NCU_TRAFFIC_BYTES.get(args.config), "kernel": "k_propagate", "kernel_ms": 1e3 * t_prop,
        "kernel_share_of_step": t_prop / (ms_step * 1e-3), "bin_kernel_ms": 1e3 * t_bin, "peak_source": peaks["source"],
        "peak_derivation": "148 SMs x 128 FP32 lanes x 2 FLOP x sm_max_mhz",
        "flop_per_photon": flop / n, "bytes_per_photon": BYTES_IN + BYTES_OUT,
        "segments_per_photon": stats["segments"] / n, "nodes_per_segment": stats["nodes"] / max(1, stats["segments"]),
        "triangle_tests_per_segment": stats["triangle_tests"] / max(1, stats["segments"]),
        "alu_tflops": alu_achieved, "alu_frac": alu_achieved / fp32_peak_tflops,
        "hbm_gbs": hbm_achieved, "hbm_frac": hbm_achieved / peaks["hbm_gbs"],
        "photons_per_s_alu_bound": n / t_alu_bound, "photons_per_s_hbm_bound": n / t_hbm_bound})
    fma = pkg.measure_fp32_peak(dev)          # FMA micro-benchmark on this device
    roof.update({"fp32_peak_measured_tflops": fma, "alu_frac_of_measured_peak": alu_achieved / fma if fma else None})

    # ---- the paper's own pipeline: filter on the efficiencies first, trace
    #      the survivors with efficiencies switched off; the survivor count never leaves the device
    paper = None
    if world == 1:
        kinds = [m["kind"] for m in w.scene.materials]
        m_mir, m_det = kinds.index(1), kinds.index(2)
        factors = [m_det] + [m_mir] * (2 if args.config in ("C4", "C5") else 1)
        pre = scene.prefilter(d_o, d_d, d_l, factors, seed=args.seed, photon_id_base=id_base, stream=stream)
        hm2, ct2 = scene.alloc_accumulators(dev)

        def paper_step(trace=True):
            hm2.zero_(); ct2.zero_()
            scene.prefilter(d_o, d_d, d_l, factors, seed=args.seed, photon_id_base=id_base, out=pre, stream=stream)
            if trace:
                scene.propagate(pre["origins"], pre["dirs"], pre["wavelengths"], seed=args.seed, records=records, hitmap=hm2,
                                counters=ct2, stream=stream, flags=pkg.FLAG_NO_EFFICIENCY, n_dev=pre["n_kept"])
        times = {}
        for name, trace in (("pipeline", True), ("prefilter", False)):
            for _ in range(args.warmup):
                paper_step(trace)
            torch.cuda.synchronize()
            ev0.record(stream)
            for _ in range(args.steps):
                paper_step(trace)
            ev1.record(stream)
            torch.cuda.synchronize()
            times[name] = ev0.elapsed_time(ev1) / args.steps * 1e-3
        kept = int(pre["n_kept"].item())
        paper_step(True)
        torch.cuda.synchronize()
        pf_bytes = 4 * n + 2 * (n // 8) + kept * (BYTES_IN + BYTES_IN + 4)      # lambda in, mask out + in, survivors in + out + index
        paper = {"what": "opx_prefilter on QE x R" + (" x R" if len(factors) == 3 else "") + " then opx_propagate_flags(NO_EFFICIENCY) on the survivors",
                 "value": n / times["pipeline"], "unit": UNIT, "ms_per_step": 1e3 * times["pipeline"],
                 "prefilter_ms": 1e3 * times["prefilter"], "kept_fraction": kept / n, "detected": int(ct2[0].item()),
                 "detected_in_flight": int(cnt[0]),
                 "prefilter_roofline": {"bound": "hbm", "achieved": pf_bytes / times["prefilter"] / 1e9, "peak": peaks["hbm_gbs"],
                                        "unit": "GB/s", "frac": pf_bytes / times["prefilter"] / 1e9 / peaks["hbm_gbs"],
                                        "bytes_per_photon": pf_bytes / n}}

    # ---- on-device Cherenkov generation from track steps, alone and chained into opx_propagate
    emit = None
    if world == 1:
        src = w.track_source if w.track_source is not None else workloads.make_config("C3", n=n).track_source
        dsteps = pkg.upload_track_steps(src.steps(), dev)
        gen = (torch.empty_like(d_o), torch.empty_like(d_d), torch.empty_like(d_l))
        hm3, ct3 = scene.alloc_accumulators(dev)

        def emit_step(trace):
            pkg.emit_cherenkov(dsteps, n, photon_id_base=0, seed=args.seed, out=gen, stream=stream)
            if trace:
                hm3.zero_(); ct3.zero_()
                scene.propagate(*gen, seed=args.seed, records=records, hitmap=hm3, counters=ct3, stream=stream)
        etimes = {}
        for name, trace in (("emit", False), ("chain", True)):
            for _ in range(args.warmup):
                emit_step(trace)
            torch.cuda.synchronize()
            ev0.record(stream)
            for _ in range(args.steps):
                emit_step(trace)
            ev1.record(stream)
            torch.cuda.synchronize()
            etimes[name] = ev0.elapsed_time(ev1) / args.steps * 1e-3
        # the paper's whole pipeline from track steps: emission fused with the filter, survivors traced with efficiencies off
        kinds_e = [m["kind"] for m in w.scene.materials]
        fac_e = [kinds_e.index(2)] + [kinds_e.index(1)] * (2 if args.config in ("C4", "C5") else 1)
        cap = n // 2 + 4096
        fpre = scene.emit_cherenkov_filtered(dsteps, n, fac_e, seed=args.seed, stream=stream, capacity=cap)
        if int(fpre["n_kept"].item()) > cap:
            raise SystemExit("bench: survivor capacity exceeded")

        def fused_step(trace):
            scene.emit_cherenkov_filtered(dsteps, n, fac_e, seed=args.seed, out=fpre, stream=stream)
            if trace:
                hm3.zero_(); ct3.zero_()
                scene.propagate(fpre["origins"], fpre["dirs"], fpre["wavelengths"], seed=args.seed,
                                records={k: v[:cap] for k, v in records.items()}, hitmap=hm3, counters=ct3, stream=stream,
                                flags=pkg.FLAG_NO_EFFICIENCY, n_dev=fpre["n_kept"])
        for name, trace in (("fused", False), ("fused_chain", True)):
            for _ in range(args.warmup):
                fused_step(trace)
            torch.cuda.synchronize()
            ev0.record(stream)
            for _ in range(args.steps):
                fused_step(trace)
            ev1.record(stream)
            torch.cuda.synchronize()
            etimes[name] = ev0.elapsed_time(ev1) / args.steps * 1e-3
        emit = {"what": f"opx_emit_cherenkov: {n} photons from {int(dsteps['length'].shape[0])} track steps"
                        + ("" if w.track_source is not None else " (step table of C3: C2's photons are a point source, not tracks)"),
                "value": n / etimes["emit"], "unit": UNIT, "ms_per_step": 1e3 * etimes["emit"],
                "roofline": {"bound": "hbm", "achieved": BYTES_IN * n / etimes["emit"] / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": BYTES_IN * n / etimes["emit"] / 1e9 / peaks["hbm_gbs"], "bytes_per_photon": BYTES_IN,
                             "note": "issue-bound on the contract's arithmetic (Philox, IEEE divides), not HBM: profiles/r01_v11_emit.md"},
                "emit_then_propagate": {"value": n / etimes["chain"], "unit": UNIT, "ms_per_step": 1e3 * etimes["chain"]},
                "emit_filtered": {"what": "opx_emit_cherenkov_filtered (emission fused with the pre-propagation filter)",
                                  "value": n / etimes["fused"], "unit": UNIT, "ms_per_step": 1e3 * etimes["fused"],
                                  "kept_fraction": int(fpre["n_kept"].item()) / n},
                "emit_filtered_then_propagate": {"what": "the paper's pipeline from track steps to hits, memory-resident: fused "
                                                         "emission + filter, survivors traced with NO_EFFICIENCY",
                                                 "value": n / etimes["fused_chain"], "unit": UNIT,
                                                 "ms_per_step": 1e3 * etimes["fused_chain"], "detected": int(ct3[0].item())}}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # bounded sample: a quick probe sets the size so that each leg is about --cpu-seconds of CPU work
        probe_n = min(n, 2000)
        rate, threads, _, _ = time_oracle(w, probe_n, args.seed)
        n_sample = int(min(n, max(probe_n, rate * args.cpu_seconds)))
        v, threads, secs, segs = time_oracle(w, n_sample, args.seed)
        n1 = int(min(n_sample, max(500, v / max(1, threads) * args.cpu_seconds)))
        v1, _, secs1, _ = time_oracle(w, n1, args.seed, n_threads=1)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"first {n_sample} photon ids of {args.config}, brute force over {w.scene.n_triangles} triangles, {secs:.1f} s "
                         f"on all cores; first {n1} ids, {secs1:.1f} s on one thread",
               "single_thread_value": v1, "ray_triangle_tests_per_s": segs * w.scene.n_triangles / secs}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"{args.config}{' + mirror vertex normals' if args.smooth else ''}: {w.scene.n_triangles} triangles, {n} photons per GPU per step "
                               f"({BYTES_IN + BYTES_OUT} B/photon = {(BYTES_IN + BYTES_OUT) * n / 1e6:.0f} MB per step)",
                   "l2": "inputs + outputs per step exceed the 126 MB L2" if (BYTES_IN + BYTES_OUT) * n > 126e6 else "fits in L2",
                   "photons_per_gpu": n, "triangles": w.scene.n_triangles, "pixels": scene.n_pixels, "seed": args.seed,
                   "id_partition": "contiguous global photon-id range per rank; scene + BVH replicated"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
        "paper_pipeline": paper, "emit": emit, "bvh_build_ms": min(t_build), "bvh_build_launches": int(build_launches),
        "states": dict(zip(pkg.STATE_NAMES, (int(x) for x in cnt[:7]))),
        "context_paper": "paper: 1.2e6 photons/s per Tesla T4 and 2e5 per Xeon thread, end to end (PAPER.md:9); other hardware, not the target",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
