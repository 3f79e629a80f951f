#!/usr/bin/env python
"""bench.py - DDF ray queries/s on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--extras]

A step = one pass of the hot path over one batch: the camera generator writes
2^20 primary rays, then ONE fused launch (rows a1-a8: load, encode, 8 layers, heads, store) answers
them.  Workload = BASELINE.json configs[1].  `value` is device-timed (CUDA events on the launching
stream, inputs resident in HBM); `e2e` goes through ddf_query_host with pinned HOST buffers.
N > 1 (torchrun): every rank runs the same per-GPU batch with its own camera (weak scaling, no
data-path collective: rays are independent, weights replicated - DESIGN.md "Multi-GPU").
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
sys.path.insert(0, ROOT)

FLOP_PER_RAY = 23_403_520            # 2*(90*1280 + 6*1280^2 + 1370*1280 + 1280*2), DESIGN.md
METRIC = "DDF ray queries/s"
UNIT = "Mrays/s"
WORKLOAD = "configs[1]: paper-scale DDF (90-dim enc, 8x1280, skip@4, bf16), 2^20 camera rays 1024x1024"
# dram__bytes_read.sum / dram__bytes_write.sum of one 2^20-ray launch of each dense kernel, from an `ncu --set full` capture:
# kept in a small text file that names its capture command and is rewritten by `bench.py --write-traffic` (below), so
# the `traffic` figures of the bench line always come from a committed artifact, never from a number typed in here.
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r03_dram_bytes.txt")


def ncu_traffic():
    """kernel name -> DRAM bytes (read + written) per launch; a kernel the file does not list reports null."""
    out = {}
    if os.path.exists(TRAFFIC_FILE):
        for line in open(TRAFFIC_FILE):
            f = line.split()
            if len(f) >= 3 and not line.startswith("#"):
                out[f[0]] = float(f[1]) + float(f[2])
    return out


def write_traffic(csv_paths, head):
    """`ncu -i X.ncu-rep --page raw --csv --print-units base > X.csv` of the capture(s) -> profiles/r03_dram_bytes.txt."""
    import csv
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    rows = {}
    for path in csv_paths:
        table = [r for r in csv.reader(open(path)) if r]
        hdr = next(i for i, r in enumerate(table) if "Kernel Name" in r)
        names, units = table[hdr], table[hdr + 1]
        ik, ir, iw = names.index("Kernel Name"), names.index("dram__bytes_read.sum"), names.index("dram__bytes_write.sum")
        for r in table[hdr + 2:]:
            kernel = r[ik].split("(")[0].split("::")[-1]
            rows[kernel] = (float(r[ir].replace(",", "")) * scale[units[ir]], float(r[iw].replace(",", "")) * scale[units[iw]])
    with open(TRAFFIC_FILE, "w") as f:
        f.write("# DRAM bytes of ONE launch on 2^20 configs[1] camera rays: kernel, dram__bytes_read.sum, dram__bytes_write.sum\n")
        f.write("# tree: %s; capture commands and the rest of the counters: profiles/r03_ncu_summary.md; written by\n" % head)
        f.write("# python bench.py --write-traffic %s\n" % " ".join(csv_paths))
        for k in sorted(rows):
            f.write("%s %.0f %.0f\n" % (k, rows[k][0], rows[k][1]))
    print(open(TRAFFIC_FILE).read())


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        j = json.load(open(p))
        return dict(burst=float(j["bf16_tflops"]), sustained=float(j.get("bf16_tflops_sustained", j["bf16_tflops"])),
                    hbm=float(j["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    return dict(burst=1590.0, sustained=1400.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        f = lambda s: float(s) if s.replace(".", "", 1).isdigit() else float("nan")
        return {"sm_mhz": statistics.median(f(r[0]) for r in rows), "sm_max_mhz": f(rows[0][1]),
                "power_w_max": max(f(r[2]) for r in rows), "samples": len(rows), "reasons": reasons}


def oracle_rate(seconds_target=12.0, mode=0):
    """rays/s of the oracle as it stands on this box's host cores, on a bounded sample of the
    configs[1] workload (camera rays through the paper-scale network)."""
    import oracle
    from ddf_inputs import MASTER_SEED, STREAMS, layout_c1, make_weights
    oracle.build()
    lay = layout_c1()
    blob = make_weights(lay)
    cam = oracle.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = oracle.gen_camera(cam, 1024, 1024)
    cores = oracle.default_threads()
    probe = max(2 * cores, 64)                               # the first call also pays for thread start-up: probe twice
    t0 = time.time(); oracle.forward(lay, blob, o[:probe], d[:probe], mode); tp = time.time() - t0
    probe2 = int(max(probe, probe * 1.5 / max(tp, 1e-3)))
    t0 = time.time(); oracle.forward(lay, blob, o[:probe2], d[:probe2], mode); tp2 = time.time() - t0
    ns = int(min(1 << 17, max(probe, probe2 * seconds_target / max(tp2, 1e-3))))
    stride = (1 << 20) // ns
    t0 = time.time(); oracle.forward(lay, blob, o[::stride][:ns], d[::stride][:ns], mode); dt = time.time() - t0
    return ns / dt, cores, "%d camera rays (every %d-th pixel of the 1024x1024 batch), %.1f s" % (ns, stride, dt)


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    rates = []
    per = max(2.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    sample = ""
    for i in range(args.warmup + args.steps):
        r, cores, sample = oracle_rate(per)
        if i >= args.warmup:
            rates.append(r)
    v = statistics.mean(rates) / 1e6
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * per, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample + " per step (CPU oracle, oracle/ddf_oracle.c, as it stands)"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def config_dict(world):
    """The workload both arms of the bench are quoted on (the reference arm times a bounded sample of it per step)."""
    return {"workload": WORKLOAD, "rays_per_gpu": 1 << 20, "parallelism": "replicas x%d, rays sharded" % world,
            "flop_per_ray": FLOP_PER_RAY, "l2": "512 MB memset between timed steps (L2 flush)",
            "step": "ddf_gen_camera + ddf_query"}


def shard_plan(world, rank, rays_per_gpu):
    """Weak scaling: every rank answers its own `rays_per_gpu` camera batch (its own seeded camera);
    no exchange step.  Returns (camera seed, first global ray index, rays)."""
    from ddf_inputs import MASTER_SEED
    return MASTER_SEED + rank, rank * rays_per_gpu, rays_per_gpu


def aggregate(times_ms_local, rays_local, dist_mod, world):
    """max-over-ranks time, sum-over-ranks rays -> whole-job Mrays/s (host logic, gloo-testable)."""
    import torch
    t = torch.tensor([float(times_ms_local)], dtype=torch.float64)
    r = torch.tensor([float(rays_local)], dtype=torch.float64)
    if world > 1:
        dev = "cuda" if dist_mod.get_backend() == "nccl" else "cpu"
        t, r = t.to(dev), r.to(dev)
        dist_mod.all_reduce(t, op=dist_mod.ReduceOp.MAX)
        dist_mod.all_reduce(r, op=dist_mod.ReduceOp.SUM)
    return float(r.item()) / float(t.item()) / 1e3, float(t.item())


def run_gpu(args):
    import torch
    import torch.distributed as dist
    import paper_2606_00817_b200 as ddf
    from ddf_inputs import STREAMS, layout_c1, layout_sdf, make_weights, random_rays

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    ddf.build()
    K, W = args.steps, max(args.warmup, 3)
    n = 1 << 20
    seed, _, _ = shard_plan(world, rank, n)
    lay = layout_c1()
    model = ddf.ddf_create(make_weights(lay), lay)
    assert ddf.ddf_get_info(model, 0) == 1
    cam = ddf.ddf_camera_from_seed(seed, STREAMS["camera_pos"], 2.5)
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
    dist_o = torch.empty(n, device="cuda"); vis_o = torch.empty(n, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")          # > 126 MB L2

    def step(ev=None):
        if ev: ev[0].record()
        ddf.ddf_gen_camera(cam, 1024, 1024, o, d)
        if ev: ev[1].record()
        ddf.ddf_query(model, o, d, n, dist_o, vis_o)
        if ev: ev[2].record()

    def timed_region():
        """W warm-up steps, then K timed steps with an L2 flush between them, clocks sampled alongside"""
        for _ in range(W):
            flush.zero_(); step()
        torch.cuda.synchronize()
        if world > 1: dist.barrier()
        torch.cuda.synchronize()
        sampler = ClockSampler(local); sampler.start(); t_wall0 = time.time()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
        for k in range(K):
            flush.zero_()                       # L2 flush between timed iterations (outside the event pairs)
            step(evs[k])
        torch.cuda.synchronize()
        if world > 1: dist.barrier()
        torch.cuda.synchronize()
        t_wall1 = time.time()
        return ([e[0].elapsed_time(e[2]) for e in evs], [e[1].elapsed_time(e[2]) for e in evs], sampler.stop(t_wall0, t_wall1))

    step_ms, kern_ms, clocks = timed_region()
    value, t_max = aggregate(sum(step_ms), n * K, dist, world)
    launches = K * 2                        # gen_camera_kernel + ddf_tc_kernel per step

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    ddf.ddf_reserve(model, ddf.RESERVE_HOST, n)       # staging sized once: no call in the timed region allocates
    oh, dh = o.cpu().pin_memory(), d.cpu().pin_memory()
    dist_h, vis_h = torch.empty(n).pin_memory(), torch.empty(n).pin_memory()
    for _ in range(2): ddf.ddf_query_host(model, oh, dh, n, dist_h, vis_h)
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    t0 = time.perf_counter()
    for _ in range(K): ddf.ddf_query_host(model, oh, dh, n, dist_h, vis_h)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_value, _ = aggregate(e2e_ms, n * K, dist, world)
    assert torch.equal(dist_h, dist_o.cpu())

    # ---- the activation-resident kernel (ddf_set_path 5) under the SAME protocol: K flushed steps, sustained clocks
    ddf.ddf_set_path(model, 5)
    _, res_kern_ms, res_clocks = timed_region()
    ddf.ddf_set_path(model, 0)

    peaks = _peaks()
    traffic = ncu_traffic()
    kern_avg = statistics.mean(kern_ms)
    achieved = n * FLOP_PER_RAY / (kern_avg * 1e-3) / 1e12
    res_avg = statistics.mean(res_kern_ms)
    res_achieved = n * FLOP_PER_RAY / (res_avg * 1e-3) / 1e12
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": t_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": config_dict(world),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 24 * n, "d2h_bytes_per_step": 8 * n},
        "gpu_launches": launches,
        "roofline": {"bound": "tensor", "kernel": "ddf_tc_kernel", "achieved": achieved, "peak": peaks["burst"],
                     "unit": "TFLOP/s", "frac": achieved / peaks["burst"], "traffic": traffic.get("ddf_tc_kernel"),
                     "frac_of_sustained_peak": achieved / peaks["sustained"], "peak_source": peaks["source"],
                     "kernel_ms": kern_avg, "kernel_share_of_step": kern_avg / statistics.mean(step_ms),
                     "ray_io_GBps": 32 * n / (kern_avg * 1e-3) / 1e9,
                     # the kernel that keeps every activation on chip, same steps, same flush, same peak
                     "resident": {"kernel": "ddf_tc_res_kernel", "kernel_ms": res_avg, "achieved": res_achieved,
                                  "frac": res_achieved / peaks["burst"], "traffic": traffic.get("ddf_tc_res_kernel"),
                                  "vs_persistent": kern_avg / res_avg, "sm_mhz": res_clocks.get("sm_mhz")}},
    }
    if rank == 0:
        if world == 1:
            r, cores, sample = oracle_rate(12.0)
            out["cpu_baseline"] = {"value": r / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        if world == 1:
            # BASELINE.json configs[2], [3], [4] in the same line (the metric is quoted "at 2^20-2^24 rays"; north_star
            # asks for the shadow / AO batches and the DDF / sphere-tracing ratio): outside the headline's timed region
            full = run_config_results(ddf, torch, model, peaks, back_to_back=args.extras)
            out["config_results"] = full if args.extras else compact_config_results(full)
        if args.extras and world == 1:
            out["extra"] = run_extras(ddf, torch, model, peaks)
        print(json.dumps(out if args.extras else sig(out)))
    if world > 1:
        dist.destroy_process_group()


def sig(x, digits=5):
    """every float of a nested result rounded to `digits` significant digits: the default line has to stay short enough
    for the driver's record to keep all of it"""
    if isinstance(x, float):
        return float("%.*g" % (digits, x)) if x == x and abs(x) != float("inf") else x
    if isinstance(x, dict):
        return {k: sig(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [sig(v, digits) for v in x]
    return x


def compact_config_results(ex):
    """The default line's copy of run_config_results: what north_star asks to be reported (camera, shadow and AO batches,
    the 2^10 .. 2^24 sweep, sphere tracing in both modes and across thresholds) without the derived fields, which follow
    from ms, the ray count and FLOP_PER_RAY.  --extras prints the long form."""
    sw = ex["sweep"]
    lgs = range(10, 25)
    st = {k[len("sphere_trace_"):]: v for k, v in ex.items() if k.startswith("sphere_trace_")}
    return sig({
        "Mrays_s": {"camera_2^20": (1 << 20) / ex["ddf_camera_2^20_ms"] / 1e3, "shadow_2^22": ex["shadow_2^22"]["Mrays_s"],
                    "ao_16.7M": ex["ao_16.7M"]["Mrays_s"]},
        "gen_ms": {"shadow_2^22": ex["shadow_2^22"]["gen_ms"], "ao_16.7M": ex["ao_16.7M"]["gen_ms"]},
        "sweep_ms_2^10..2^24": [sw["2^%d" % lg]["ms"] for lg in lgs],
        "sweep_ms_back_to_back_2^10..2^17": [sw["2^%d" % lg]["ms_back_to_back"] for lg in range(10, 18)],
        # [ms, MLP evaluations, DDF speed-up] per tracer mode / hit threshold
        "sphere_trace_ms_evals_ddfx": {k: [v["ms"], v["mlp_evals"], v["ddf_speedup"]] for k, v in st.items()},
    }, 4)


def _time_ms(torch, fn, reps=3, warm=1):
    for _ in range(warm): fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); fn(); e1.record(); torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    return statistics.median(ts)


def run_config_results(ddf, torch, model, peaks, back_to_back=False):
    """The other BASELINE.json configs, each measured the same way (CUDA events on the launching stream, median of 3
    after 1 warm-up, inputs resident): shadow (configs[2]), AO with the on-GPU reduction (configs[3]), the batch
    sweep 2^10 .. 2^24 and the sphere-tracing comparison on the camera rays (configs[4])."""
    from ddf_inputs import MASTER_SEED, STREAMS, layout_sdf, make_weights, random_rays
    ex = {}
    tf = lambda n, ms: n * FLOP_PER_RAY / (ms * 1e-3) / 1e12
    # ---- configs[2]: shadow rays
    n = 1 << 22
    p = torch.empty((n, 3), device="cuda"); nr = torch.empty((n, 3), device="cuda")
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda"); tm = torch.empty(n, device="cuda")
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    gen_ms = _time_ms(torch, lambda: (ddf.ddf_gen_sphere_points(MASTER_SEED, STREAMS["shadow_points"], n, 1.0, p, nr),
                                      ddf.ddf_gen_shadow(p, nr, n, (3.0, 3.0, 3.0), 1e-3, o, d, tm)))
    q_ms = _time_ms(torch, lambda: ddf.ddf_query(model, o, d, n, dist, vis))
    ex["shadow_2^22"] = {"query_ms": q_ms, "Mrays_s": n / q_ms / 1e3, "TFLOPs": tf(n, q_ms), "frac_peak": tf(n, q_ms) / peaks["burst"],
                         "gen_ms": gen_ms, "gen_GBps": (n * 24 + n * 52) / (gen_ms * 1e-3) / 1e9}
    del p, nr, tm
    # ---- configs[3]: AO, 1024x1024 x 16 spp, reduced on the GPU inside the query kernel
    W = H = 1024; npts = W * H; spp = 16; n = npts * spp
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    sc = ddf.DdfScene((0.0, 0.0, 0.0), 0.6, (-3.0, -3.0, -3.0), (3.0, 3.0, 3.0))
    gp = torch.empty((npts, 3), device="cuda"); gn = torch.empty((npts, 3), device="cuda")
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda"); ao = torch.empty(npts, device="cuda")
    gen_ms = _time_ms(torch, lambda: (ddf.ddf_gen_gbuffer(cam, sc, W, H, gp, gn, None),
                                      ddf.ddf_gen_ao(gp, gn, npts, spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3, o, d)))
    q_ms = _time_ms(torch, lambda: ddf.ddf_query_ao(model, o, d, npts, spp, float("inf"), ao), reps=2)
    ex["ao_16.7M"] = {"query_ao_ms": q_ms, "Mrays_s": n / q_ms / 1e3, "TFLOPs": tf(n, q_ms), "frac_peak": tf(n, q_ms) / peaks["burst"],
                      "gen_ms": gen_ms, "gen_GBps": (n * 24 + npts * 24 * 2) / (gen_ms * 1e-3) / 1e9,
                      "gen_frac_hbm": (n * 24 + npts * 24 * 2) / (gen_ms * 1e-3) / 1e9 / peaks["hbm"]}
    # ---- configs[4]: batch sweep 2^10 .. 2^24 (prefixes of the AO ray buffer, incoherent rays)
    sweep = {}
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    for lg in range(10, 25):
        m = 1 << lg
        ms = _time_ms(torch, lambda: ddf.ddf_query(model, o, d, m, dist, vis), reps=3 if lg > 20 else 7)
        sweep["2^%d" % lg] = {"ms": ms, "ns_per_ray": ms * 1e6 / m, "Mrays_s": m / ms / 1e3, "frac_peak": tf(m, ms) / peaks["burst"]}
        if lg <= 17:      # an isolated call on an idle stream above (latency); here the per-call time of calls queued back to back (throughput)
            nb = (50 if lg <= 14 else 16) if back_to_back else (20 if lg <= 14 else 8)
            def burst():
                for _ in range(nb): ddf.ddf_query(model, o, d, m, dist, vis)
            bb = _time_ms(torch, burst, reps=3) / nb
            sweep["2^%d" % lg]["ms_back_to_back"] = bb
            sweep["2^%d" % lg]["frac_peak_back_to_back"] = tf(m, bb) / peaks["burst"]
    ex["sweep"] = sweep
    del o, d, dist, vis, ao
    # ---- configs[4]: sphere tracing an SDF MLP of the same width and depth on the camera rays
    n = 1 << 20
    lay = layout_sdf()
    sdf = ddf.ddf_create(make_weights(lay), lay)
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, 1024, 1024, o, d)
    t = torch.empty(n, device="cuda"); hit = torch.empty(n, dtype=torch.uint8, device="cuda")
    st = torch.empty(n, dtype=torch.int32, device="cuda"); tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    ddf_ms = _time_ms(torch, lambda: ddf.ddf_query(model, o, d, n, dist, vis))
    SDF_FLOP = 23_262_720
    for name, early in (("fixed64", 0), ("early_exit", 1)):
        prm = ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, early)
        ms = _time_ms(torch, lambda: ddf.sdf_sphere_trace(sdf, o, d, n, prm, t, hit, st, None, None, tot), reps=2)
        evals = int(tot.item())
        ex["sphere_trace_" + name] = {"ms": ms, "Mrays_s": n / ms / 1e3, "mlp_evals": evals, "mean_steps": float(st.float().mean()),
                                      "hit_rate": float(hit.float().mean()), "TFLOPs": evals * SDF_FLOP / (ms * 1e-3) / 1e12,
                                      "frac_peak": evals * SDF_FLOP / (ms * 1e-3) / 1e12 / peaks["burst"], "ddf_speedup": ms / ddf_ms}
    # "across convergence thresholds": the early-exit tracer at two more hit thresholds
    for eps in (1e-2, 1e-4):
        prm = ddf.SdfTraceParams(64, eps, 6.0, 1.0, 0.05, 1)
        ms = _time_ms(torch, lambda: ddf.sdf_sphere_trace(sdf, o, d, n, prm, t, hit, st, None, None, tot), reps=2)
        ex["sphere_trace_early_exit_eps%g" % eps] = {"ms": ms, "mlp_evals": int(tot.item()), "mean_steps": float(st.float().mean()),
                                                     "hit_rate": float(hit.float().mean()), "ddf_speedup": ms / ddf_ms}
    ex["ddf_camera_2^20_ms"] = ddf_ms
    ddf.ddf_destroy(sdf)
    # ---- the same camera batch on the activation-resident kernel (ddf_set_path 5): no activation leaves the SM pair
    ddf.ddf_set_path(model, 5)
    res_ms = _time_ms(torch, lambda: ddf.ddf_query(model, o, d, n, dist, vis), reps=5)
    ddf.ddf_set_path(model, 0)
    ex["resident_kernel_camera_2^20"] = {"ms": res_ms, "Mrays_s": n / res_ms / 1e3, "TFLOPs": tf(n, res_ms), "frac_peak": tf(n, res_ms) / peaks["burst"],
                                         "vs_persistent_kernel": ddf_ms / res_ms, "dram_traffic_bytes_ncu": ncu_traffic().get("ddf_tc_res_kernel"),
                                         "persistent_kernel_dram_traffic_bytes_ncu": ncu_traffic().get("ddf_tc_kernel")}
    return ex


def run_extras(ddf, torch, model, peaks):
    """--extras: the SURVEY.md 8(f) rows (hash-grid field, wavefront, training, narrow networks)."""
    from ddf_inputs import MASTER_SEED, STREAMS, layout_sdf, make_weights
    ex = {}
    ex["sphere_trace_relaxation"] = run_relaxation_table(ddf, torch, model)
    ex["hashgrid_field"] = run_hashgrid(ddf, torch, peaks)
    ex["wavefront_shadowed_camera_2^20"] = run_wavefront(ddf, torch)
    ex["training_hashgrid"] = run_training(ddf, torch)
    ex["training_hashgrid_fp32_cuda_cores"] = run_training(ddf, torch, arithmetic=1)
    ex["narrow_networks_2^20_random_rays"] = run_narrow(ddf, torch)
    return ex


def run_relaxation_table(ddf, torch, model):
    """SURVEY.md 8(f) f4 / PAPER.md:112 ("across ray counts and across convergence thresholds"), Table IV: the early-exit
    sphere tracer with plain (omega 1) and over-relaxed steps on three views of the same SDF network - head-on from
    radius 2.5 (the configs[4] view), grazing (a 10-degree view aimed at the limb of the unit sphere, every ray within 5
    degrees of the tangent), close and off-axis (radius 1.2, looking past the centre) - at three hit thresholds.
    Per cell: [ms, MLP evaluations, hit rate, DDF speed-up] on 2^18 rays (512 x 512); DDF time = one ddf_query of the batch."""
    from ddf_inputs import MASTER_SEED, STREAMS, layout_sdf, make_weights
    lay = layout_sdf()
    sdf = ddf.ddf_create(make_weights(lay), lay)
    W = H = 512; n = W * H
    head = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    px, py, pz = [float(x) for x in head.pos]
    r = (px * px + py * py + pz * pz) ** 0.5
    ux, uy, uz = px / r, py / r, pz / r                          # towards the camera
    # any unit vector normal to u: the limb point of the unit sphere seen from distance r is u / r + sqrt(1 - 1/r^2) v
    ax = (0.0, 0.0, 1.0) if abs(uz) < 0.9 else (1.0, 0.0, 0.0)
    vx, vy, vz = uy * ax[2] - uz * ax[1], uz * ax[0] - ux * ax[2], ux * ax[1] - uy * ax[0]
    vn = (vx * vx + vy * vy + vz * vz) ** 0.5
    vx, vy, vz = vx / vn, vy / vn, vz / vn
    c = (1.0 - 1.0 / (r * r)) ** 0.5
    limb = (ux / r + c * vx, uy / r + c * vy, uz / r + c * vz)
    views = {
        "head_on_r2.5_fov50": ddf.DdfCamera(head.pos, (0.0, 0.0, 0.0), 50.0),
        "grazing_r2.5_fov10_at_limb": ddf.DdfCamera(head.pos, limb, 10.0),
        "off_axis_r1.2_fov50": ddf.DdfCamera((1.2 * ux, 1.2 * uy, 1.2 * uz), (0.8 * vx, 0.8 * vy, 0.8 * vz), 50.0),
    }
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
    t = torch.empty(n, device="cuda"); hit = torch.empty(n, dtype=torch.uint8, device="cuda")
    st = torch.empty(n, dtype=torch.int32, device="cuda"); tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    out = {}
    for name, cam in views.items():
        ddf.ddf_gen_camera(cam, W, H, o, d)
        ddf_ms = _time_ms(torch, lambda: ddf.ddf_query(model, o, d, n, dist, vis))
        cell = {"ddf_ms": ddf_ms}
        for eps in (1e-2, 1e-3, 1e-4):
            for omega in (1.0, 1.2, 1.6):
                prm = ddf.SdfTraceParams(64, eps, 6.0, 1.0, 0.05, 1, omega)
                ms = _time_ms(torch, lambda: ddf.sdf_sphere_trace(sdf, o, d, n, prm, t, hit, st, None, None, tot), reps=2)
                cell["eps%g_omega%g" % (eps, omega)] = [ms, int(tot.item()), float(hit.float().mean()), ms / ddf_ms]
        out[name] = cell
    ddf.ddf_destroy(sdf)
    return sig(out, 4)


def run_narrow(ddf, torch):
    """BASELINE.json configs[0] (3 x 64, 54-dim input) and the paper's own sinusoidal MLPs of its encoding
    ablation (128 x 4 and 256 x 6; band counts as configs[1]) on 2^20 random rays.
    Widths 64 / 128 run on the shared-memory-resident tcgen05 kernel (ddf_narrow.cu), 256 on the
    persistent kernel of the headline config."""
    from ddf_inputs import Layout, layout_c0, make_weights, random_rays, blob_layer_shapes
    n = 1 << 20
    o_np, d_np = random_rays(n)
    o = torch.from_numpy(o_np).cuda(); d = torch.from_numpy(d_np).cuda()
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    out = {}
    for name, lay in (("configs[0]_64x3", layout_c0()), ("paper_128x4", Layout(0, 10, 4, 4, 128, -1, 2, 0)),
                      ("paper_256x6", Layout(0, 10, 4, 6, 256, -1, 2, 0))):
        m = ddf.ddf_create(make_weights(lay), lay)
        ms = _time_ms(torch, lambda: ddf.ddf_query(m, o, d, n, dist, vis), reps=7)
        flop = 2 * sum(a * b for a, b in blob_layer_shapes(lay))
        out[name] = {"ms": ms, "Mrays_s": n / ms / 1e3, "TFLOPs": n * flop / (ms * 1e-3) / 1e12, "flop_per_ray": flop,
                     "launches": ddf.ddf_get_info(m, 1), "tcgen05": ddf.ddf_get_info(m, 0)}
        ddf.ddf_set_path(m, 1)
        ms1 = _time_ms(torch, lambda: ddf.ddf_query(m, o, d, n, dist, vis), reps=3)
        out[name]["cuda_core_path_ms"] = ms1
        ddf.ddf_destroy(m)
    return out


def run_training(ddf, torch, steps=30000, batch=16384, arithmetic=0):
    """the paper's recipe (Adam, 30,000 steps, batch 16,384, lr 3e-3 with
    cosine decay to 5 %, clamped L1 + 0.3 CE, 30 % ray-march shifted samples) on an ANALYTIC scene (a
    sphere over a slab; the paper's scanned objects are not in the container), then the paper-style
    end metrics of the trained field against the analytic ray caster (its stand-in for Embree):
    primary-ray depth error / hit agreement and shadow-ray agreement.  The
    paper's own training time is quoted as context: "under an hour" on one A100."""
    from ddf_inputs import MASTER_SEED, STREAMS, layout_hash_paper, make_hash_table, make_hash_mlp
    lay = layout_hash_paper()
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table, mlp = make_hash_table(lay, n_ent, scale=1e-4), make_hash_mlp(lay)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(total_steps=steps, arithmetic=arithmetic))
    scene = ddf.DdfScene((0.0, 0.0, 0.0), 0.5, (-0.9, -0.9, -0.9), (0.9, 0.9, -0.6))
    o = torch.empty((batch, 3), device="cuda"); d = torch.empty((batch, 3), device="cuda")
    t = torch.empty(batch, device="cuda"); hit = torch.empty(batch, dtype=torch.uint8, device="cuda")
    losses = torch.zeros(steps, device="cuda")
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for s in range(steps):
        ddf.ddf_gen_train_batch(scene, MASTER_SEED, STREAMS["train_rays"], s, batch, 2.9, o, d, t, hit)
        ddf.ddf_trainer_step(tr, o, d, t, hit, batch, losses[s:s + 1])
    e1.record(); torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) / 1e3
    l = losses.cpu().numpy()
    out = {"arithmetic": ["bf16x3 tensor cores", "fp32 CUDA cores"][arithmetic], "steps": steps, "batch": batch, "seconds": sec, "steps_per_s": steps / sec, "Mrays_per_s": steps * batch / sec / 1e6,
           "loss_first_100": float(l[:100].mean()), "loss_last_100": float(l[-100:].mean()),
           "paper_context": "30,000 steps x 16,384 rays in under an hour on one A100 (PAPER.md:86), PyTorch"}
    tt, mm = ddf.ddf_trainer_export(tr, 2 * n_ent, len(mlp))
    ddf.ddf_trainer_destroy(tr)
    m = ddf.ddf_create_hashgrid(tt, mm, lay)
    # ---- end metrics, ground truth = the analytic ray caster
    dist = torch.empty(batch, device="cuda"); vis = torch.empty(batch, device="cuda")
    ddf.ddf_gen_train_batch(scene, MASTER_SEED, STREAMS["train_rays"], 10 ** 6, batch, 2.9, o, d, t, hit)     # held-out batch
    ddf.ddf_query(m, o, d, batch, dist, vis)
    hh = hit > 0
    out["heldout_hit_agreement"] = float(((vis > 0.5) == hh).float().mean())
    out["heldout_depth_mae_on_hits"] = float((dist - t).abs()[hh].mean())
    out["heldout_depth_median_abs_err"] = float((dist - t).abs()[hh].median())
    # secondary rays from an analytic G-buffer (the paper's use: PAPER.md:80, 155): 512 x 512 view, light (3,3,3)
    W = H = 512; n = W * H
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    po = torch.empty((n, 3), device="cuda"); pd = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, W, H, po, pd)
    gt_t = torch.empty(n, device="cuda"); gt_h = torch.empty(n, dtype=torch.uint8, device="cuda")
    ddf.ddf_scene_raycast(scene, po, pd, n, gt_t, gt_h)
    pix = torch.nonzero(gt_h > 0).flatten()
    k = int(pix.numel())
    light = torch.tensor((3.0, 3.0, 3.0), device="cuda")
    so = (po[pix] + (gt_t[pix] - 2e-3)[:, None] * pd[pix]).contiguous()
    sd = light[None, :] - so; tmax = sd.norm(dim=1); sd = (sd / tmax[:, None]).contiguous()
    st = torch.empty(k, device="cuda"); sh = torch.empty(k, dtype=torch.uint8, device="cuda")
    ddf.ddf_scene_raycast(scene, so, sd, k, st, sh)
    gt_shadow = (sh > 0) & (st < tmax)
    d2 = torch.empty(k, device="cuda"); v2 = torch.empty(k, device="cuda"); ds = torch.empty(k, dtype=torch.uint8, device="cuda")
    ddf.ddf_query(m, so, sd, k, d2, v2)
    ddf.ddf_shadow_test(v2, d2, tmax, k, ds)
    out["shadow_ray_agreement"] = float(((ds > 0) == gt_shadow).float().mean())
    out["shadow_fraction_ground_truth"] = float(gt_shadow.float().mean())
    mse = float((((ds > 0).float() - gt_shadow.float()) ** 2).mean())
    out["shadow_mask_psnr_db"] = float(-10.0 * np.log10(max(mse, 1e-12)))
    # ambient occlusion over the same G-buffer: 16 cosine samples per pixel, "average the hit flag"
    gp = (po[pix] + gt_t[pix][:, None] * pd[pix]).contiguous()
    on_sphere = (gp.norm(dim=1) - 0.5).abs() < 1e-4
    bmin = torch.tensor((-0.9, -0.9, -0.9), device="cuda"); bmax = torch.tensor((0.9, 0.9, -0.6), device="cuda")
    dlo, dhi = (gp - bmin[None, :]).abs(), (gp - bmax[None, :]).abs()
    face = torch.cat([dlo, dhi], dim=1).argmin(dim=1)                     # 0..2: min faces, 3..5: max faces
    gn = torch.zeros_like(gp)
    gn[torch.arange(k, device="cuda"), face % 3] = torch.where(face < 3, -1.0, 1.0)
    gn[on_sphere] = gp[on_sphere] / gp[on_sphere].norm(dim=1, keepdim=True)
    gn = gn.contiguous()
    spp = 16
    ao_o = torch.empty((k * spp, 3), device="cuda"); ao_d = torch.empty((k * spp, 3), device="cuda")
    ddf.ddf_gen_ao(gp, gn, k, spp, MASTER_SEED, STREAMS["ao_samples"], 2e-3, ao_o, ao_d)
    at = torch.empty(k * spp, device="cuda"); ah = torch.empty(k * spp, dtype=torch.uint8, device="cuda")
    ddf.ddf_scene_raycast(scene, ao_o, ao_d, k * spp, at, ah)
    ao_gt = 1.0 - ah.view(k, spp).float().mean(dim=1)
    ao = torch.empty(k, device="cuda")
    ddf.ddf_query_ao(m, ao_o, ao_d, k, spp, float("inf"), ao)
    out["ao_mae"] = float((ao - ao_gt).abs().mean())
    out["ao_psnr_db"] = float(-10.0 * np.log10(max(float(((ao - ao_gt) ** 2).mean()), 1e-12)))
    out["ao_mean_ground_truth"] = float(ao_gt.mean())
    out["paper_context_metrics"] = "shadows 30.3 dB, AO 21.3 dB, AO MAE 0.216 over 142 scanned objects vs Embree (PAPER.md:248-256)"
    # primary rays from the camera itself (one shared origin: only the 27-dim direction code varies)
    pdist = torch.empty(n, device="cuda"); pvis = torch.empty(n, device="cuda")
    ddf.ddf_query(m, po, pd, n, pdist, pvis)
    gh = gt_h > 0
    out["primary_hit_agreement"] = float(((pvis > 0.5) == gh).float().mean())
    out["primary_depth_mae_on_common_hits"] = float((pdist - gt_t).abs()[gh & (pvis > 0.5)].mean())
    out["view"] = "512x512 pinhole at radius 2.5, %d of %d pixels hit" % (k, n)
    # the same frame with NO analytic G-buffer ("no mesh in the pipeline"): hit points and normals from
    # the field's own primary answers, shadow + AO rays from there (ddf_query_shaded), judged against the scene
    lit = torch.empty(n, dtype=torch.uint8, device="cuda"); nrm = torch.empty((n, 3), device="cuda")
    aow = torch.empty(n, device="cuda"); cs = torch.zeros(2, dtype=torch.int64, device="cuda")
    eps_w = 2e-2
    ddf.ddf_query_shaded(m, po, pd, W, H, [(3.0, 3.0, 3.0)], spp, MASTER_SEED, STREAMS["ao_samples"], eps_w, float("inf"),
                         pdist, pvis, lit, nrm, aow, cs)
    both = gh & (pvis > 0.5)
    gn_img = torch.zeros((n, 3), device="cuda"); gn_img[pix] = gn
    ang = torch.rad2deg(torch.acos((nrm * gn_img).sum(1)[both].clamp(-1.0, 1.0)))
    gs_img = torch.zeros(n, dtype=torch.bool, device="cuda"); gs_img[pix] = gt_shadow
    mf = {"eps": eps_w, "pixels_hit_by_both": int(both.sum().item()),
          "normal_error_deg_median": float(ang.median()), "normal_error_deg_mean": float(ang.mean()),
          "shadow_agreement": float(((lit == 0) == gs_img)[both].float().mean())}
    # AO: the scene ray-cast along the very rays the wavefront traced (isolates the field's answers from sampling noise)
    p_c = torch.empty((n, 3), device="cuda"); n_c = torch.empty((n, 3), device="cuda"); idx = torch.empty(n, dtype=torch.int32, device="cuda")
    wo = torch.empty((n * spp, 3), device="cuda"); wd = torch.empty((n * spp, 3), device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    ddf.ddf_gen_ao_from_hits(m, po, pd, pdist, pvis, W, H, spp, MASTER_SEED, STREAMS["ao_samples"], eps_w, p_c, n_c, idx, wo, wd, cnt)
    kk = int(cnt.item())
    wt = torch.empty(kk * spp, device="cuda"); wh = torch.empty(kk * spp, dtype=torch.uint8, device="cuda")
    ddf.ddf_scene_raycast(scene, wo[:kk * spp].contiguous(), wd[:kk * spp].contiguous(), kk * spp, wt, wh)
    ao_scene = 1.0 - wh.view(kk, spp).float().mean(dim=1)
    ao_field = aow[idx[:kk].long()]
    mf["ao_mae_same_rays"] = float((ao_field - ao_scene).abs().mean())
    ao_gt_img = torch.ones(n, device="cuda"); ao_gt_img[pix] = ao_gt
    mf["ao_mae_vs_gbuffer_ao_other_samples"] = float((aow - ao_gt_img).abs()[both].mean())
    mf["rays"] = {"shadow": int(cs[0].item()), "ao": int(cs[1].item())}
    out["meshfree_frame"] = mf
    ddf.ddf_destroy(m)
    return out


def run_wavefront(ddf, torch):
    """primary query -> hit compaction -> shadow rays -> second query -> lit flags in
    one call (ddf_query_shadowed) on the 2^20 camera batch with spread origins; visibility-head bias 1
    so that most rays hit.  Rays/s counts primary + secondary evaluations."""
    from ddf_inputs import MASTER_SEED, STREAMS, layout_c1, layout_hash_paper, make_weights, make_hash_table, make_hash_mlp, random_rays
    out = {}
    n = 1 << 20
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, 1024, 1024, o, d)
    o += torch.from_numpy(random_rays(n)[0]).cuda() * 0.4
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    lit = torch.empty(n, dtype=torch.uint8, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    lay = layout_c1(); blob = make_weights(lay).copy(); blob[-1] = 0x3F80
    hl = layout_hash_paper(); mlp = make_hash_mlp(hl).copy(); mlp[-1] = 1.0
    models = {"dense_8x1280": ddf.ddf_create(blob, lay),
              "hashgrid": ddf.ddf_create_hashgrid(make_hash_table(hl, ddf.ddf_hashgrid_table_entries(hl)), mlp, hl)}
    for name, m in models.items():
        ms = _time_ms(torch, lambda: ddf.ddf_query_shadowed(m, o, d, n, (3.0, 3.0, 3.0), 1e-3, dist, vis, lit, cnt), reps=5)
        k = int(cnt.item())
        out[name] = {"ms": ms, "shadow_rays": k, "lit_fraction_of_hits": float(lit.sum().item()) / max(k, 1),
                     "launches": ddf.ddf_get_info(m, 1), "Mrays_s_primary_plus_secondary": (n + k) / ms / 1e3}
        # three point lights from the same hit points (ddf_query_shadowed_lights): one primary query, three shadow queries
        lights = [(3.0, 3.0, 3.0), (-3.0, 2.0, 1.0), (0.5, -4.0, 2.5)]
        ms3 = _time_ms(torch, lambda: ddf.ddf_query_shadowed_lights(m, o, d, n, lights, 1e-3, dist, vis, lit, cnt), reps=5)
        k3 = int(cnt.item())
        out[name]["three_lights"] = {"ms": ms3, "shadow_rays": k3, "launches": ddf.ddf_get_info(m, 1),
                                     "Mrays_s_primary_plus_secondary": (n + k3) / ms3 / 1e3}
        # ambient occlusion at the field's own hits (ddf_query_ao_wavefront): normals from the hit-point image,
        # 16 cosine-weighted rays per hit, fused reduce; 1024 x 1024 primary rays
        ao = torch.empty(n, device="cuda")
        msa = _time_ms(torch, lambda: ddf.ddf_query_ao_wavefront(m, o, d, 1024, 1024, 16, MASTER_SEED, STREAMS["ao_samples"], 1e-3,
                                                                 float("inf"), dist, vis, None, ao, cnt), reps=3)
        ka = int(cnt.item())
        out[name]["ao_16spp"] = {"ms": msa, "ao_rays": ka, "mean_ao_of_hits": float(ao[vis > 0.5].mean().item()),
                                 "launches": ddf.ddf_get_info(m, 1), "Mrays_s_primary_plus_secondary": (n + ka) / msa / 1e3}
        ddf.ddf_destroy(m)
    return out


def run_hashgrid(ddf, torch, peaks):
    """the paper's own field (hash grid 16 x 2 x 2^19 + 4 direction bands + 2 x 64
    MLP, 52 MB fp32) on the same batch shapes.  Bound: 128 random 8-byte gathers per ray (one 32-byte
    sector each) served by L1/L2; `gather_GBps` counts the 1024 B/ray actually used, `sector_GBps`
    the 4096 B/ray of sectors moved.  The paper's own figure for this field (tiny-cuda-nn on an
    A100) is quoted as context only."""
    from ddf_inputs import MASTER_SEED, STREAMS, layout_hash_paper, make_hash_table, make_hash_mlp, random_rays
    lay = layout_hash_paper()
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table, mlp = make_hash_table(lay, n_ent), make_hash_mlp(lay)
    m = ddf.ddf_create_hashgrid(table, mlp, lay)
    out = {"table_entries": n_ent, "field_MB": (2 * n_ent + 8130) * 4 / 1e6,
           "paper_context": {"Mrays_s": 333.0, "what": "tiny-cuda-nn, A100, 1M rays (PAPER.md:202: 0.0030 us/ray)"}}
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)

    def rec(name, n, ms):
        out[name] = {"ms": ms, "Mrays_s": n / ms / 1e3, "gather_GBps": n * 1024 / (ms * 1e-3) / 1e9,
                     "sector_GBps": n * 4096 / (ms * 1e-3) / 1e9}
    n = 1 << 22
    o_np, d_np = random_rays(n)
    o = torch.from_numpy(o_np).cuda() * 2.9; d = torch.from_numpy(d_np).cuda()
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    rec("random_origins_2^22", n, _time_ms(torch, lambda: ddf.ddf_query(m, o, d, n, dist, vis), reps=7))
    for lg in (10, 14, 18):
        k = 1 << lg
        rec("random_origins_2^%d" % lg, k, _time_ms(torch, lambda: ddf.ddf_query(m, o, d, k, dist, vis), reps=7))
    oc = torch.empty((1 << 20, 3), device="cuda"); dc = torch.empty((1 << 20, 3), device="cuda")
    ddf.ddf_gen_camera(cam, 1024, 1024, oc, dc)
    rec("camera_2^20", 1 << 20, _time_ms(torch, lambda: ddf.ddf_query(m, oc, dc, 1 << 20, dist, vis), reps=7))
    # the same frame through ddf_query_camera: rays generated in the kernel, origin features once per CTA
    rec("camera_2^20_fused_generator", 1 << 20, _time_ms(torch, lambda: ddf.ddf_query_camera(m, cam, 1024, 1024, dist, vis), reps=7))
    p = torch.empty((n, 3), device="cuda"); nr = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_sphere_points(MASTER_SEED, STREAMS["shadow_points"], n, 1.0, p, nr)
    ddf.ddf_gen_shadow(p, nr, n, (3.0, 3.0, 3.0), 1e-3, o, d, None)
    rec("shadow_2^22", n, _time_ms(torch, lambda: ddf.ddf_query(m, o, d, n, dist, vis), reps=7))
    del p, nr, o, d
    W = H = 1024; npts = W * H; spp = 16; na = npts * spp
    sc = ddf.DdfScene((0.0, 0.0, 0.0), 0.6, (-3.0, -3.0, -3.0), (3.0, 3.0, 3.0))
    gp = torch.empty((npts, 3), device="cuda"); gn = torch.empty((npts, 3), device="cuda")
    ddf.ddf_gen_gbuffer(cam, sc, W, H, gp, gn, None)
    oa = torch.empty((na, 3), device="cuda"); da = torch.empty((na, 3), device="cuda"); ao = torch.empty(npts, device="cuda")
    ddf.ddf_gen_ao(gp, gn, npts, spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3, oa, da)
    rec("ao_16.7M_fused", na, _time_ms(torch, lambda: ddf.ddf_query_ao(m, oa, da, npts, spp, float("inf"), ao), reps=5))
    # the same AO image from the G-buffer points themselves (ddf_query_ao_points): rays generated inside the kernel
    ao_pts = torch.empty(npts, device="cuda")
    rec("ao_16.7M_from_points", na, _time_ms(torch, lambda: ddf.ddf_query_ao_points(m, gp, gn, npts, spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3,
                                                                                        float("inf"), ao_pts), reps=5))
    out["ao_16.7M_from_points"]["bit_identical_to_gen_plus_query_ao"] = bool(torch.equal(ao, ao_pts))
    del oa, da
    ddf.ddf_destroy(m)
    # the same field with an fp16 table (26 MB): random origins again
    from ddf_inputs import HashLayout
    lay16 = HashLayout(table_dtype=2)
    m16 = ddf.ddf_create_hashgrid(make_hash_table(lay16, n_ent), mlp, lay16)
    o = torch.from_numpy(o_np).cuda() * 2.9; d = torch.from_numpy(d_np).cuda()
    rec("random_origins_2^22_fp16_table", n, _time_ms(torch, lambda: ddf.ddf_query(m16, o, d, n, dist, vis), reps=7))
    ddf.ddf_destroy(m16)
    del o, d
    # the oracle on the host cores, bounded sample
    import oracle
    k = 1 << 17
    t0 = time.time(); oracle.hash_forward(lay, table, mlp, o_np[:k] * 2.9, d_np[:k]); dt = time.time() - t0
    out["cpu_oracle"] = {"Mrays_s": k / dt / 1e6, "cores": oracle.default_threads(), "sample": "%d random-origin rays, %.2f s" % (k, dt)}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--extras", action="store_true", help="also measure shadow / AO / sweep / sphere tracing")
    ap.add_argument("--write-traffic", nargs="+", metavar="NCU_RAW_CSV",
                    help="no benchmark: rewrite profiles/r03_dram_bytes.txt from `ncu --page raw --csv --print-units base` files")
    args = ap.parse_args()
    if args.write_traffic:
        head = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
        write_traffic(args.write_traffic, "commit " + head if head else "unknown commit")
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
