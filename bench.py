#!/usr/bin/env python
"""bench.py -- photons/s of the per-photon optical propagation hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C4] [--photons n]

One "step" = one opx_propagate call (ONE kernel: staging, sort, traversal, interaction, records, hit binning and
counters) over one batch of synthetic photons, inputs resident in HBM.  The headline line is on the largest
single-GPU configuration of BASELINE.json, C4 = configs[3]: the LHCb-RICH-like scene (1.01e6 triangles, meshes at
5 mm) with 1e8 track photons per step.  The other configurations (C1, C2, C3 on
the toy scene, the C5 stream on the C4 scene) are timed in the same run and reported as sub-records under
"configs", each with its own roofline fraction.  The BVH build is timed separately (`bvh_build_ms`, SURVEY.md
8(d)).  N > 1 (torchrun): every rank propagates its own contiguous id range of the same size (weak scaling) and the
per-rank hit-maps and counters are summed with one NCCL all-reduce per step.  Prints ONE JSON line on rank 0.
"""
import argparse
import concurrent.futures
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
BYTES_IN, BYTES_OUT = 28, 34                        # per photon: inputs, hit record
L2_BYTES = 126e6                                    # replaced by the device's own L2 size in main() (device_constants)
N_SMS = 148                                         # likewise: the device's SM count


def device_constants(torch, dev):
    """L2 size and SM count of the device the bench runs on (they decide how small configs are timed and the derived peak)."""
    global L2_BYTES, N_SMS
    prop = torch.cuda.get_device_properties(dev)
    L2_BYTES = float(getattr(prop, "L2_cache_size", 0) or L2_BYTES)
    N_SMS = int(prop.multi_processor_count)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the step's kernel, from the `ncu --set full` captures
# summarised under profiles/ (per config, at the launch size this bench times; None until a capture exists)
NCU_TRAFFIC_BYTES = {"C2": (565296128, 10_000_000), "C4": (6683452000, 100_000_000)}      # (bytes, photons of the captured launch)
NCU_TRAFFIC_SOURCE = {"C2": "profiles/r02_k_propagate_packet.md (1e7 photons per launch)", "C4": "profiles/r02_k_propagate_packet.md (1e8 photons per launch)"}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


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
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))
        except Exception:
            pass

    def stop(self, t0=None, t1=None):
        """Summary of the samples taken in [t0, t1] (perf_counter; all samples if None)."""
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=2)
        rows = [r for t, r in self.rows if (t0 is None or t >= t0) and (t1 is None or t <= t1)]
        sm = [float(r[0]) for r in rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = sorted({names[k] for r in rows if len(r) >= 7 for k in range(4) if r[3 + k].startswith("Active")})
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    power_w_max=max(pw) if pw else None, reasons=reasons, samples=len(sm))


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


def workload_name(name, scene, n, smooth=False):
    return (f"{name}{' + mirror vertex normals' if smooth else ''}: {scene.n_triangles} triangles, {n} photons per GPU per step "
            f"({BYTES_IN + BYTES_OUT} B/photon = {(BYTES_IN + BYTES_OUT) * n / 1e6:.0f} MB per step)")


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
    po, pd, pl = w.photon_range(0, 200)
    t0 = time.perf_counter()
    oracle.trace_mesh(w.scene, po, pd, pl, seed=args.seed)
    rate = 200 / (time.perf_counter() - t0)
    n_sample = int(min(w.n, args.reference_sample, max(200, rate * 3.0)))
    o, d, lam = w.photon_range(0, n_sample)
    for _ in range(args.warmup):
        oracle.trace_mesh(w.scene, o[:200], d[:200], lam[:200], seed=args.seed)
    t0 = time.perf_counter()
    threads = 0
    for _ in range(args.steps):
        r = oracle.trace_mesh(w.scene, o, d, lam, seed=args.seed)
        threads = r["n_threads"]
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = f"first {n_sample} photon ids of {args.config} per step, brute force over {w.scene.n_triangles} triangles"
    n_full = min(w.n, 100_000_000)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.config, w.scene, n_full, args.smooth) + " (the oracle runs a bounded sample of it)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def pinned_photons(w, id_base, n, threads=8):
    """The workload's photons id_base .. id_base + n - 1 in pinned host tensors (generated in slices, in parallel:
    every photon is a pure function of (seed, id))."""
    import torch
    pin = [torch.empty((n, 3), dtype=torch.float32).pin_memory(), torch.empty((n, 3), dtype=torch.float32).pin_memory(),
           torch.empty(n, dtype=torch.float32).pin_memory()]
    step = 2_000_000

    def fill(a):
        b = min(n, a + step)
        for dst, src in zip(pin, w.photon_range(id_base + a, id_base + b)):
            dst[a:b] = torch.from_numpy(src)
    with concurrent.futures.ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(fill, range(0, n, step)))
    return pin


class Timed:
    """Device timing of `steps` calls of step() on `stream` (CUDA events around the whole region; when the step's
    working set fits in L2 every step is timed on its own with an L2 flush -- a 256 MB fill -- before it)."""

    def __init__(self, torch, stream, dev):
        self.torch, self.stream, self.dev = torch, stream, dev
        self.flush_buf = None

    def run(self, step, steps, warmup, flush_l2=False):
        torch = self.torch
        for _ in range(warmup):
            step()
        torch.cuda.synchronize()
        if not flush_l2:
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record(self.stream)
            for _ in range(steps):
                step()
            ev1.record(self.stream)
            torch.cuda.synchronize()
            return ev0.elapsed_time(ev1)
        if self.flush_buf is None:
            self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            self.flush_buf.fill_(1)
            a.record(self.stream)
            step()
            b.record(self.stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs)


def roofline_record(pkg, scene, photons, n, id_base, seed, kernel_ms, step_ms, peaks, fma_peak, config, kernel_ms_all=None):
    """algorithmic FLOPs (instrumented single-ray walk: segments, node visits, triangle tests,
    interactions) and bytes (62 B/photon) of one launch over the kernel's measured duration; the slower bound is named."""
    d_o, d_d, d_l = photons
    stats = scene.propagate_stats(d_o, d_d, d_l, seed=seed, photon_id_base=id_base)
    flop = (FLOP_NODE * stats["nodes"] + FLOP_TRI * stats["triangle_tests"] + FLOP_SEGMENT * stats["segments"]
            + FLOP_INTERACTION * stats["interactions"])
    t = kernel_ms * 1e-3
    derived = N_SMS * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    peak = fma_peak if fma_peak else derived
    alu = flop / t / 1e12
    hbm_bytes = (BYTES_IN + BYTES_OUT) * n
    hbm = hbm_bytes / t / 1e9
    t_alu, t_hbm = flop / (peak * 1e12), hbm_bytes / (peaks["hbm_gbs"] * 1e9)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": alu, "peak": peak, "unit": "TFLOP/s", "frac": alu / peak,
                "peak_source": "measured (FP32 FMA micro-benchmark opx_measure_fp32_peak on this device)" if fma_peak
                               else f"derived ({N_SMS} SMs x 128 FP32 lanes x 2 FLOP x sm_max_mhz)"}
    else:
        roof = {"bound": "hbm", "achieved": hbm, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": hbm / peaks["hbm_gbs"],
                "peak_source": peaks["source"]}
    roof.update({
        # the capture's bytes, scaled when this launch has another photon count than the captured one (the default sizes match)
        "traffic": (NCU_TRAFFIC_BYTES[config][0] * n // NCU_TRAFFIC_BYTES[config][1]) if config in NCU_TRAFFIC_BYTES else None,
        "traffic_source": NCU_TRAFFIC_SOURCE.get(config),
        # not a measurement of THIS run: the bytes of an earlier ncu capture (a run under ncu is never a bench run)
        "traffic_measured_in_run": False,
        "traffic_scaled_from_capture": bool(config in NCU_TRAFFIC_BYTES and n != NCU_TRAFFIC_BYTES[config][1]),
        "kernel": pkg.last_kernel(), "kernel_ms": kernel_ms, "kernel_share_of_step": kernel_ms / step_ms,
        # median and best of the per-launch times next to the mean the fractions above use
        "kernel_ms_median": statistics.median(kernel_ms_all) if kernel_ms_all else None,
        "kernel_ms_best": min(kernel_ms_all) if kernel_ms_all else None,
        "kernel_ms_launches": len(kernel_ms_all) if kernel_ms_all else 0,
        "fp32_peak_derived_tflops": derived, "frac_of_derived_peak": alu / derived,
        "fp32_peak_derivation": f"{N_SMS} SMs x 128 FP32 lanes x 2 FLOP x sm_max_mhz (only the clock is measured)",
        "flop_per_photon": flop / n, "bytes_per_photon": BYTES_IN + BYTES_OUT,
        "segments_per_photon": stats["segments"] / n, "nodes_per_segment": stats["nodes"] / max(1, stats["segments"]),
        "triangle_tests_per_segment": stats["triangle_tests"] / max(1, stats["segments"]),
        "alu_tflops": alu, "hbm_gbs": hbm, "hbm_frac": hbm / peaks["hbm_gbs"], "hbm_peak_source": peaks["source"],
        "photons_per_s_alu_bound": n / t_alu, "photons_per_s_hbm_bound": n / t_hbm})
    return roof


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
                         "kernel": pkg.last_kernel(), "gpu_launches": pkg.launch_count() - l0})
    best = max(rows, key=lambda r: r["photons_per_s"])
    print(json.dumps({"metric": METRIC, "value": best["photons_per_s"], "unit": UNIT, "n_gpus": 1, "higher_is_better": True,
                      "dtype": "f32", "data": "synthetic", "scaling": "weak", "vs_baseline": None,
                      "config": {"workload": f"{args.config} chunk-size sweep: {w.scene.n_triangles} triangles, resident batch of {n} photons "
                                             f"streamed until {args.total} photons per chunk size", "best_chunk": best["chunk"]},
                      "sweep": rows}))


def sub_record(pkg, torch, tm, name, dev, seed, peaks, fma_peak, target_s, n=None, workload=None):
    """One of the other BASELINE.json configurations, device-timed in this run: value, ms/step, roofline.
    A configuration whose inputs + outputs fit in L2 (C1, the paper's 6e5-photon run) is timed as a STREAM of calls over K
    distinct resident batches (consecutive ids of the same workload) whose inputs + outputs together exceed twice the L2, so
    that no step finds its photons in L2 while the scene stays warm -- what a caller streaming chunks sees."""
    import workloads
    w = workload if workload is not None else workloads.make_config(name, n=n)
    n = w.n
    small = (BYTES_IN + BYTES_OUT) * n <= L2_BYTES
    K = int(np.ceil(2 * L2_BYTES / ((BYTES_IN + BYTES_OUT) * n))) if small else 1
    if K > 1:
        # the same workload with K x n photons: batch k = ids [k n, (k+1) n)
        w = workloads.make_config(w.name, n=K * n)
    scene = pkg.Scene(w.scene).build(dev)
    batches = []
    for k in range(K):
        pin = pinned_photons(w, k * n, n)
        batches.append((tuple(x.to(dev, non_blocking=True) for x in pin), scene.alloc_records(n, dev)))
    torch.cuda.synchronize()
    photons = batches[0][0]
    hitmap, counters = scene.alloc_accumulators(dev)
    it = [0]

    def step():
        ph, rec = batches[it[0] % K]
        hitmap.zero_(); counters.zero_()
        scene.propagate(*ph, seed=seed, photon_id_base=(it[0] % K) * n, records=rec, hitmap=hitmap, counters=counters, stream=tm.stream)
        it[0] += 1
    ms = tm.run(step, 3 * K if K > 1 else 3, 2)
    steps = int(min(4000, max(5, target_s / max(1e-6, ms / (3 * K if K > 1 else 3) * 1e-3))))
    if K > 1:
        steps = (steps + K - 1) // K * K
    for _ in range(3):
        step()
    it[0] = 0
    scene.profile_begin(steps)
    l0 = pkg.launch_count()
    ms_total = tm.run(step, steps, 0, flush_l2=False)
    launches = pkg.launch_count() - l0
    ms_prop, _ = scene.profile_end()
    kernel_ms = statistics.mean(ms_prop)
    ms_step = ms_total / steps
    # counters of the last step (batch K-1)
    cnt = counters.cpu().numpy()
    roof = roofline_record(pkg, scene, batches[(steps - 1) % K][0], n, ((steps - 1) % K) * n, seed, kernel_ms, ms_step, peaks, fma_peak, name, ms_prop)
    return {"workload": workload_name(name, w.scene, n), "value": n / (ms_step * 1e-3), "unit": UNIT, "steps": steps,
            "ms_per_step": ms_step, "gpu_launches": int(launches),
            "l2": (f"a stream of calls over {K} distinct resident batches ({K * (BYTES_IN + BYTES_OUT) * n / 1e6:.0f} MB of inputs + outputs, "
                   f"twice the {L2_BYTES / 1e6:.0f} MB L2): no step finds its photons in L2, the scene stays warm") if K > 1 else f"inputs + outputs per step exceed the {L2_BYTES / 1e6:.0f} MB L2",
            "roofline": roof, "states": dict(zip(pkg.STATE_NAMES, (int(x) for x in cnt[:7])))}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="opx", choices=["opx", "reference"])
    ap.add_argument("--config", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--photons", type=int, default=None, help="photons per GPU per step (default: the config's N, at most 1e8)")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="CPU time budget of each cpu_baseline leg (all cores, one thread)")
    ap.add_argument("--reference-sample", type=int, default=20000)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sub-records", action="store_true", help="skip the C1/C2/C3/C5 sub-records, the paper pipeline and the emission legs")
    ap.add_argument("--sub-seconds", type=float, default=0.25, help="length of the timed region of each sub-record")
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
    device_constants(torch, dev)
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
    ranks = [{"rank": rank, "id_base": int(id_base), "photons": int(n), "device": torch.cuda.get_device_name(dev)}]
    if dist is not None:
        gathered = [None] * world
        dist.all_gather_object(gathered, ranks[0])
        ranks = gathered
        if rank == 0:      # what a cold N > 1 run is: communicator size and each rank's id range, before anything is timed
            print(f"[bench] world {world}, NCCL communicator of {dist.get_world_size()} ranks: " +
                  "; ".join(f"rank {r['rank']} ids [{r['id_base']}, {r['id_base'] + r['photons']})" for r in ranks), file=sys.stderr)
    # the ranks of one node generate their photons side by side: share the host cores instead of 8 threads each
    gen_threads = max(1, min(8, (os.cpu_count() or 8) // max(1, world)))
    pin = pinned_photons(w, id_base, n, threads=gen_threads)
    d_o, d_d, d_l = (x.to(dev, non_blocking=True) for x in pin)
    stream = torch.cuda.current_stream(dev)
    tm = Timed(torch, stream, dev)

    # ---- scene + BVH build (timed separately: SURVEY.md 8(d))
    scene = pkg.Scene(w.scene)
    scene.build(dev)
    l0 = pkg.launch_count()
    torch.cuda.synchronize()
    t_build = []
    for _ in range(3):
        t0 = time.perf_counter()
        scene.build(dev)
        t_build.append(1e3 * (time.perf_counter() - t0))
    build_launches = (pkg.launch_count() - l0) // 3

    records = scene.alloc_records(n, dev)
    if args.sweep:
        hitmap, counters = scene.alloc_accumulators(dev)
        return run_sweep(args, scene, (d_o, d_d, d_l), records, hitmap, counters, n, stream, w, pkg)

    # ---- the headline: exactly --steps timed calls, barrier + synchronize on both sides, max over ranks
    hitmap, counters = scene.alloc_accumulators(dev)

    def step():
        hitmap.zero_(); counters.zero_()
        scene.propagate(d_o, d_d, d_l, seed=args.seed, photon_id_base=id_base, records=records, hitmap=hitmap,
                        counters=counters, stream=stream)
        allreduce_accumulators(hitmap, counters)                      # the one exchange step (no-op at N = 1)

    flush = (BYTES_IN + BYTES_OUT) * n <= L2_BYTES
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    scene.profile_begin(args.steps)
    l0 = pkg.launch_count()
    torch.cuda.synchronize()
    t_begin = time.perf_counter()
    ms_total = tm.run(step, args.steps, 0, flush_l2=flush)
    t_end = time.perf_counter()
    if dist is not None:
        dist.barrier()
    launches = pkg.launch_count() - l0                           # kernels of libopx.so only (torch fills not counted)
    ms_prop, _ = scene.profile_end()
    kernel_name = pkg.last_kernel()
    clocks = sampler.stop(t_begin, t_end)
    clocks["timed_region_s"] = t_end - t_begin
    if dist is not None:
        t = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = world * n * args.steps / (ms_total * 1e-3)
    cnt = counters.cpu().numpy()

    # ---- end to end through the C ABI with host buffers (copies inside the timed region).  The headline form returns what the
    #      paper asks for: the list of DETECTED photons + hit-map + counters; `records` is the same call returning
    #      every photon's 34-byte record; `tracks` starts from the track steps in host memory, so that the photons
    #      never cross the link at all.
    e2e = None
    if rank == 0 or dist is not None:
        def wall(fn, k):
            fn()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(k):
                fn()
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            if dist is not None:
                t = torch.tensor([dt], device=dev, dtype=torch.float64)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                dt = float(t.item())
            return dt / k
        chunk = min(n, 1 << 21)
        cap = max(4096, int(1.25 * int(cnt[0])) + 4096)
        host_det = pkg.alloc_host_detected(cap, scene.n_pixels)

        def e2e_step():
            host_det["hitmap"].zero_(); host_det["counters"].zero_()
            scene.propagate_host_detected(*pin, seed=args.seed, photon_id_base=id_base, chunk=chunk, out=host_det, stream=stream)
        dt = wall(e2e_step, args.e2e_steps)
        n_det = int(host_det["n_detected"])
        e2e = {"value": world * n / dt, "unit": UNIT, "h2d_bytes_per_step": BYTES_IN * n,
               "d2h_bytes_per_step": 36 * n_det + 4 * scene.n_pixels + 72, "chunk_photons": chunk, "ms_per_step": 1e3 * dt,
               "detected_per_step": n_det,
               "what": "opx_propagate_host_detected: pinned host photon arrays in (28 B/photon), the list of detected photons "
                       "(id, pixel, position, direction: 36 B each) + hit-map + counters out"}
        if dist is None and (n_det != int(cnt[0]) or not np.array_equal(host_det["counters"].numpy(), cnt)):
            raise SystemExit("bench: host path and device path disagree")
        del host_det
        if dist is None:
            host_out = pkg.alloc_host_records(n, scene.n_pixels)
            chunk_r = min(n, 1 << 20)

            def rec_step():
                host_out["hitmap"].zero_(); host_out["counters"].zero_()
                scene.propagate_host(*pin, seed=args.seed, photon_id_base=id_base, chunk=chunk_r, out=host_out, stream=stream)
            dt = wall(rec_step, args.e2e_steps)
            e2e["records"] = {"value": n / dt, "unit": UNIT, "h2d_bytes_per_step": BYTES_IN * n,
                              "d2h_bytes_per_step": BYTES_OUT * n + 4 * scene.n_pixels + 64, "chunk_photons": chunk_r, "ms_per_step": 1e3 * dt,
                              "what": "opx_propagate_host: the same with every photon's 34-byte hit record brought back"}
            if not np.array_equal(host_out["counters"].numpy(), cnt):
                raise SystemExit("bench: host record path and device path disagree")
            del host_out
            if w.track_source is not None and id_base == 0:
                # the step table in page-locked host memory, like the photon arrays of the other legs
                steps_h = {k: torch.from_numpy(v).pin_memory().numpy() for k, v in w.track_source.steps().items()}
                kinds_ = [m["kind"] for m in w.scene.materials]
                fac_ = [kinds_.index(2)] + [kinds_.index(1)] * (2 if args.config in ("C4", "C5") else 1)
                tr = {}
                for name, fac in (("in_flight", ()), ("paper_filter", fac_)):
                    hd = pkg.alloc_host_detected(cap, scene.n_pixels)
                    dt = wall(lambda: scene.tracks_host_detected(steps_h, n, factors=fac, seed=args.seed, out=hd, chunk=min(n, 1 << 26), stream=stream),
                              args.e2e_steps)
                    tr[name] = {"value": n / dt, "unit": UNIT, "ms_per_step": 1e3 * dt, "detected_per_step": int(hd["n_detected"]),
                                "h2d_bytes_per_step": 40 * len(steps_h["length"]) + 8, "d2h_bytes_per_step": 36 * int(hd["n_detected"]) + 4 * scene.n_pixels + 72}
                    del hd
                e2e["tracks"] = dict(tr, what="opx_tracks_host_detected: track steps in host memory in (40 B/step), photons generated and "
                                              "propagated on the device, list of detected photons out; in_flight = efficiencies drawn per "
                                              "interaction, paper_filter = the paper's pre-propagation filter fused with the emission")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, DESIGN.md section 9
    peaks = measured_peaks()
    fma = pkg.measure_fp32_peak(dev)          # FMA micro-benchmark on this device
    pkg_kernel = kernel_name
    roof = roofline_record(pkg, scene, (d_o, d_d, d_l), n, id_base, args.seed, statistics.mean(ms_prop), ms_step, peaks, fma, args.config, ms_prop)
    roof["kernel"] = pkg_kernel

    paper = emit = None
    subs = {}
    if world == 1 and not args.no_sub_records:
        # ---- the paper's own pipeline: filter on the efficiencies first, trace
        #      the survivors with efficiencies switched off; the survivor count never leaves the device
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
        k_sub = max(3, min(args.steps, 10))
        times = {name: tm.run(lambda: paper_step(trace), k_sub, args.warmup) / k_sub * 1e-3
                 for name, trace in (("pipeline", True), ("prefilter", False))}
        kept = int(pre["n_kept"].item())
        paper_step(True)
        torch.cuda.synchronize()
        pf_bytes = 4 * n + 2 * (n // 8) + kept * (BYTES_IN + BYTES_IN + 4)      # lambda in, mask out + in, survivors in + out + index
        paper = {"what": "opx_prefilter on QE x R" + (" x R" if len(factors) == 3 else "") + " then opx_propagate_flags(NO_EFFICIENCY) on the survivors",
                 "value": n / times["pipeline"], "unit": UNIT, "ms_per_step": 1e3 * times["pipeline"],
                 "prefilter_ms": 1e3 * times["prefilter"], "kept_fraction": kept / n, "detected": int(ct2[0].item()),
                 "detected_in_flight": int(cnt[0]), "trace_kernel": pkg.last_kernel(),
                 "prefilter_roofline": {"bound": "hbm", "achieved": pf_bytes / times["prefilter"] / 1e9, "peak": peaks["hbm_gbs"],
                                        "unit": "GB/s", "frac": pf_bytes / times["prefilter"] / 1e9 / peaks["hbm_gbs"],
                                        "bytes_per_photon": pf_bytes / n}}
        del pre

        # ---- on-device Cherenkov generation from track steps, alone and chained into opx_propagate
        src = w.track_source if w.track_source is not None else workloads.make_config("C3", n=n).track_source
        dsteps = pkg.upload_track_steps(src.steps(), dev)
        gen = (torch.empty_like(d_o), torch.empty_like(d_d), torch.empty_like(d_l))
        hm3, ct3 = scene.alloc_accumulators(dev)

        def emit_step(trace):
            pkg.emit_cherenkov(dsteps, n, photon_id_base=0, seed=args.seed, out=gen, stream=stream)
            if trace:
                hm3.zero_(); ct3.zero_()
                scene.propagate(*gen, seed=args.seed, records=records, hitmap=hm3, counters=ct3, stream=stream)
        etimes = {name: tm.run(lambda: emit_step(trace), k_sub, args.warmup) / k_sub * 1e-3
                  for name, trace in (("emit", False), ("chain", True))}
        # the paper's whole pipeline from track steps: emission fused with the filter, survivors traced with efficiencies off
        cap = n // 2 + 4096
        fpre = scene.emit_cherenkov_filtered(dsteps, n, factors, seed=args.seed, stream=stream, capacity=cap)
        if int(fpre["n_kept"].item()) > cap:
            raise SystemExit("bench: survivor list truncated (capacity)")

        def fused_step(trace):
            scene.emit_cherenkov_filtered(dsteps, n, factors, seed=args.seed, out=fpre, stream=stream)
            if trace:
                hm3.zero_(); ct3.zero_()
                scene.propagate(fpre["origins"], fpre["dirs"], fpre["wavelengths"], seed=args.seed,
                                records={k: v[:cap] for k, v in records.items()}, hitmap=hm3, counters=ct3, stream=stream,
                                flags=pkg.FLAG_NO_EFFICIENCY, n_dev=fpre["n_kept"])
        for name, trace in (("fused", False), ("fused_chain", True)):
            etimes[name] = tm.run(lambda: fused_step(trace), k_sub, args.warmup) / k_sub * 1e-3
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
        del gen, fpre

        # ---- the C5 stream on this scene (BASELINE.json configs[4]): photons of C5's tracks (beta in [0.9999, 1], disc
        #      radius 200 mm) generated ON THE DEVICE from its step table, streamed in chunks with advancing ids
        if args.config in ("C4", "C5"):
            n5 = n
            w5 = workloads.make_config("C5", n=n5)
            st5 = pkg.upload_track_steps(w5.track_source.steps(), dev)
            g5 = pkg.emit_cherenkov(st5, n5, photon_id_base=0, seed=args.seed, stream=stream)
            hm5, ct5 = scene.alloc_accumulators(dev)
            passes = [0]

            def c5_step():
                scene.propagate(*g5, seed=args.seed, photon_id_base=passes[0] * n5, records=records, hitmap=hm5, counters=ct5, stream=stream)
                passes[0] += 1
            k5 = max(3, min(args.steps, 10))
            ms5 = tm.run(c5_step, k5, args.warmup) / k5
            subs["C5"] = {"workload": f"C5 stream: {w.scene.n_triangles} triangles, {k5} chunks of {n5} photons (of the 1e9-photon stream; ids continue "
                                      f"across chunks), photons generated on the device by opx_emit_cherenkov from C5's step table",
                          "value": n5 / (ms5 * 1e-3), "unit": UNIT, "steps": k5, "ms_per_step": ms5, "kernel": pkg.last_kernel(),
                          "hbm_gbs_algorithmic": n5 * (BYTES_IN + BYTES_OUT) / (ms5 * 1e-3) / 1e9,
                          "note": "chunk-size sweep 1e5..1e8 with ncu counters: `bench.py --config C5 --sweep`, profiles/r02_c5_sweep.md"}
            del g5
        del records
        torch.cuda.empty_cache()
        # ---- the other configurations, each device-timed here with its own roofline
        for name in ("C1", "C2", "C3"):
            if name != args.config:
                subs[name] = sub_record(pkg, torch, tm, name, dev, args.seed, peaks, fma, args.sub_seconds)
        # the paper's own run size (600 ... 6e5 photons per run) on the headline scene
        w6 = workloads.make_config(args.config if args.config in ("C4", "C5") else "C4", n=600_000)
        subs["paper_run_6e5"] = sub_record(pkg, torch, tm, "C4 scene, the paper's largest run (6e5 photons, PAPER.md:175)", dev, args.seed,
                                           peaks, fma, args.sub_seconds, workload=w6)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # bounded sample: a quick probe sets the size so that each leg is about --cpu-seconds of CPU work
        probe_n = min(n, 400)
        rate, threads, _, _ = time_oracle(w, probe_n, args.seed)
        n_sample = int(min(n, max(probe_n, rate * args.cpu_seconds)))
        v, threads, secs, segs = time_oracle(w, n_sample, args.seed)
        n1 = int(min(n_sample, max(100, v / max(1, threads) * args.cpu_seconds)))
        v1, _, secs1, _ = time_oracle(w, n1, args.seed, n_threads=1)
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"first {n_sample} photon ids of {args.config}, brute force over {w.scene.n_triangles} triangles, {secs:.1f} s "
                         f"on all cores; first {n1} ids, {secs1:.1f} s on one thread",
               "single_thread_value": v1, "ray_triangle_tests_per_s": segs * w.scene.n_triangles / secs}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, w.scene, n, args.smooth),
                   "l2": "every step timed on its own after a 256 MB fill that flushes L2" if flush else f"inputs + outputs per step exceed the {L2_BYTES / 1e6:.0f} MB L2",
                   "photons_per_gpu": n, "triangles": w.scene.n_triangles, "pixels": scene.n_pixels, "seed": args.seed,
                   "id_partition": "contiguous global photon-id range per rank; scene + BVH replicated",
                   "ranks": [[r["id_base"], r["photons"]] for r in ranks]},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
        "configs": subs, "paper_pipeline": paper, "emit": emit, "bvh_build_ms": min(t_build), "bvh_build_launches": int(build_launches),
        "states": dict(zip(pkg.STATE_NAMES, (int(x) for x in cnt[:7]))),
        "context_paper": "paper: 1.2e6 photons/s per Tesla T4 and 2e5 per Xeon thread, end to end (PAPER.md:9); other hardware, not the target",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
