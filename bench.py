#!/usr/bin/env python
"""bench.py — TPC cluster finder on B200: digits/s (BASELINE.json:metric) on a synthetic time frame.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--path fused|general] [--impl reference]

A step = one pass of the whole hot path (SURVEY.md §8(a) K0..K5 = one tpc_cf_run) over one full time frame that is
already resident in HBM.  Default workload: BASELINE.json configs[2] (36 sectors x 152 rows x 138 pads x 14336 time
bins, ~2 % occupancy, seed 3) — the full frame the north_star's target is quoted on; it fits one GPU.
N > 1 (torchrun): replicas only ("avoiding any GPU intercommunication"): every rank
processes its own frame (frame index = rank), no data-path collective; value = total digits / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/, as it stands, single thread) on a bounded sample of the same
workload on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "tpc_digits_per_second"
UNIT = "digits/s"


def load_peaks():
    """Measured roofline denominators (driver-written), else the fallback of B200_PROFILING.md."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def load_traffic(workload, path, kernel):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture, or None (also None
    when the capture is of another kernel than the one that ran)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(p) as f:
            t = json.load(f)
        e = t.get("%s/%s" % (workload, path))
        return float(e["dram_bytes_per_launch"]) if e and e.get("kernel") == kernel else None
    except Exception:
        return None


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe): one
    `nvidia-smi -lms` process streams a line every 20 ms; only lines stamped inside [enter, exit] are kept."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.all_rows = []
        self.proc = None
        self.th = None
        self.t0 = self.t1 = None

    def start(self):
        """Launch the sampler early (it needs ~0.5 s to come up); __enter__/__exit__ mark the timed region."""
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return self

        def pump():
            for line in self.proc.stdout:
                self.all_rows.append((time.perf_counter(), [c.strip() for c in line.strip().split(",")]))
        self.th = threading.Thread(target=pump, daemon=True)
        self.th.start()
        return self

    def __enter__(self):
        if self.proc is None and self.th is None:
            self.start()
        self.t0 = time.perf_counter()
        return self

    def __exit__(self, *a):
        self.t1 = time.perf_counter()
        time.sleep(0.05)
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=3)
            except Exception:
                self.proc.kill()
        inside = [r for (t, r) in self.all_rows if self.t0 <= t <= self.t1 + 0.03 and len(r) >= 7]
        near = [r for (t, r) in self.all_rows if len(r) >= 7]
        self.rows = inside if inside else near[-3:]

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows), "power_w_max": max(pw) if pw else None}


def oracle_sample(cfg_id, n_sectors_sample, frame=0):
    """Bounded sample for the CPU oracle: the first n_sectors_sample sectors of the workload (same bytes as the
    full frame's slice).  Returns (digits, geometry)."""
    from datagen import gen
    geom = gen.geometry(cfg_id)
    d = gen.generate(cfg_id, frame=frame, sectors=(0, n_sectors_sample))
    return d, geom


def time_oracle(digits, geom, n_sectors_sample):
    from oracle import oracle as orc
    t0 = time.perf_counter()
    cl, st = orc.run(digits, geom[0], geom[1], geom[2], geom[3], npads=geom[4],
                     planes=(0, n_sectors_sample * geom[1]))
    dt = time.perf_counter() - t0
    return dt, st


def sample_sectors(cfg_id, per_step=False):
    # measured ~2 ms per 138x14336 plane single-threaded (config 3): the whole frame is ~11 s (config 4 ~28 s), which
    # is the cpu_baseline sample; the --impl reference arm times 8 sectors per step (~2.5 s) so that K + W steps
    # end within minutes.  config 1/2 have one sector.
    from datagen import gen
    return min(gen.CONFIGS[cfg_id]["n_sectors"], 8 if per_step else 36)


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    if args.stage in ("fe", "ec"):
        return run_reference_stage(args)
    from datagen import gen
    from oracle import oracle as orc
    orc.build()
    ns = sample_sectors(args.config, per_step=True)
    digits, geom = oracle_sample(args.config, ns)
    for _ in range(min(args.warmup, 1)):
        time_oracle(digits, geom, ns)
    times = []
    for _ in range(args.steps):
        dt, st = time_oracle(digits, geom, ns)
        times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = digits.shape[0] / (ms * 1e-3)
    sample = "first %d of %d sectors of the frame (%d digits, %d clusters) per step" % (
        ns, geom[0], digits.shape[0], st["n_clusters"])
    line = {"metric": METRIC, "value": value, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u16/i64/f64", "data": "synthetic",
            "config": {"workload": "config%d: %s" % (args.config, gen.CONFIGS[args.config]["label"]),
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "clusters_per_s": st["n_clusters"] / (ms * 1e-3)}
    print(json.dumps(line))
    return 0


def run_reference_stage(args):
    """--impl reference --stage fe|ec: that stage's oracle, as it stands, single thread, on a bounded sample of the
    same workload per step (fe: the raw samples of the first sector; ec: the first ~2 M clusters of the oracle cluster
    finder's output on the first 8 sectors)."""
    from datagen import gen
    cfg = dict(gen.CONFIGS[args.config])
    if args.stage == "fe":
        from datagen import fe_gen
        from oracle import fe_oracle as feo
        feo.build()
        ns, nr, mp, nt, npads = gen.geometry(cfg)
        d = gen.generate(cfg, sectors=(0, 1))
        raw, ped4 = fe_gen.raw_from_digits(d, ns, nr, mp, nt, npads=npads, seed=cfg["seed"], planes=(0, nr))
        units = (int(np.sum(npads)) if npads is not None else nr * mp) * nt
        fn = lambda: feo.run(raw, ped4, 1, nr, mp, nt, npads=npads, zs_threshold=3)
        metric, unit = "tpc_raw_samples_filtered_per_second", "samples/s"
        sample = "raw samples of the first sector (%d valid samples) per step" % units
    else:
        from oracle import oracle as orc, ec_oracle as eco
        orc.build(); eco.build()
        ns = min(cfg["n_sectors"], 8)
        geom = gen.geometry(cfg)
        d = gen.generate(cfg, sectors=(0, ns))
        cl, _ = orc.run(d, geom[0], geom[1], geom[2], geom[3], npads=geom[4], planes=(0, ns * geom[1]))
        units = int(cl.shape[0])
        fn = lambda: eco.encode(cl, geom[0], geom[1])
        metric, unit = "tpc_clusters_encoded_per_second", "clusters/s"
        sample = "the %d clusters of the first %d sectors per step" % (units, ns)
    for _ in range(min(args.warmup, 1)):
        fn()
    times = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        fn()
        times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(times))
    value = units / (ms * 1e-3)
    line = {"metric": metric, "value": value, "unit": unit, "impl": "reference", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "i64", "data": "synthetic",
            "config": {"workload": "%s stage on config%d: %s" % (args.stage, args.config, cfg["label"]), "sample": sample},
            "cpu_baseline": {"value": value, "unit": unit, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def run_ec(args):
    """--stage ec: the entropy coder (include/tpc_ec.h) on the cluster stream of one frame of the chosen config, as
    the chain of PAPER.md:57 has it: the cluster finder's output is coded on the device without leaving it.  One GPU.
    A step = one tpc_ec_encode (all its kernels); the decoder is timed the same way and reported beside it."""
    import torch
    from datagen import gen
    import paper_2402_01205_b200 as cf
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    dev = "cuda:0"
    torch.cuda.set_device(0)
    cfg = gen.CONFIGS[args.config]
    geom = gen.geometry(args.config)
    digits = gen.generate(args.config)
    nd = int(digits.shape[0])
    finder = cf.ClusterFinder(*geom[:4], npads=geom[4], max_digits=nd, max_clusters=nd // 10 + 1024, device=dev)
    d = cf.to_device(digits)
    finder.run(d, nd, flags=cf.DIGITS_SORTED)
    cl_host, st = finder.result()
    n = st["n_clusters"]
    clusters = finder.clusters[:n * 32].clone()
    del d
    finder.close()
    del finder
    torch.cuda.empty_cache()
    coder = cf.ClusterCoder(geom[0], geom[1], n, device=dev)
    out = torch.empty(coder.max_encoded_bytes(n), dtype=torch.uint8, device=dev)
    back = torch.empty(n * 32, dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2, written between timed calls

    def timed(fn, steps):
        ms = []
        for _ in range(steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        return ms

    enc = lambda: coder.encode(clusters, n, out)
    sampler = ClockSampler(0).start()
    timed(enc, args.warmup)
    est = coder.read_status()
    if est["error"]:
        raise RuntimeError("encode failed: %r" % (est,))
    total = est["bytes"]
    enc_launches = coder.last_launch_count()
    dec = lambda: coder.decode(out, total, n, back)
    timed(dec, args.warmup)
    dst = coder.read_status()
    if dst["error"]:
        raise RuntimeError("decode failed: %r" % (dst,))
    dec_launches = coder.last_launch_count()
    with sampler as clocks:
        enc_ms = timed(enc, args.steps)
        dec_ms = timed(dec, args.steps)
    e_ms, d_ms = float(np.mean(enc_ms)), float(np.mean(dec_ms))
    # integer fields must survive the round trip bit-exactly (the floats are quantised by the format)
    b = back.cpu().numpy().view(cf.CLUSTER)
    for fld in ("sector", "row", "pad", "time", "qmax", "qtot", "flags"):
        if not np.array_equal(b[fld], cl_host[fld]):
            raise RuntimeError("round trip changed field %s" % fld)
    peak, peak_src = load_peaks()
    # algorithmic bytes of one encode: 32 B/cluster read + 13 B/cluster symbol streams written and read twice
    # (histogram, coder) + the container written; DESIGN.md §10
    alg = 32.0 * n + 13.0 * n * 3 + float(total)
    host_out = torch.empty(out.numel(), dtype=torch.uint8, pin_memory=True)
    host_in = torch.from_numpy(cl_host.view(np.uint8)).pin_memory()
    dev_in = torch.empty(n * 32, dtype=torch.uint8, device=dev)

    def e2e_step():
        dev_in.copy_(host_in, non_blocking=True)
        coder.encode(dev_in, n, out)
        s = coder.read_status()
        host_out[:s["bytes"]].copy_(out[:s["bytes"]], non_blocking=True)
        torch.cuda.synchronize()
    e2e_step()
    t0 = time.perf_counter()
    for _ in range(3):
        e2e_step()
    x_ms = (time.perf_counter() - t0) * 1e3 / 3
    line = {"metric": "tpc_clusters_encoded_per_second", "value": n / (e_ms * 1e-3), "unit": "clusters/s",
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": e_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u8/u32", "data": "synthetic",
            "config": {"workload": "entropy coder (TPC-EC v1) on the cluster stream of config%d: %s" % (
                           args.config, cfg["label"]), "stage": "ec", "clusters": n, "container_bytes": total,
                       "bits_per_cluster": 8.0 * total / n, "ratio_vs_32B_records": 32.0 * n / total,
                       "l2": "256 MB written between timed calls (L2 flush)"},
            "decode": {"ms": d_ms, "clusters_per_s": n / (d_ms * 1e-3), "gpu_launches": dec_launches},
            "roofline": {"bound": "hbm", "kernel": "tpc_ec_encode (all %d kernels)" % enc_launches,
                         "achieved": alg / (e_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s", "peak_source": peak_src,
                         "frac": alg / (e_ms * 1e-3) / 1e9 / peak, "traffic": None,
                         "algorithmic_bytes_per_launch": alg,
                         "note": "the coder is bound by the serial rANS recurrence per lane (ALU latency), not by HBM"},
            "cpu_baseline": None,
            "e2e": {"value": n / (x_ms * 1e-3), "unit": "clusters/s", "ms_per_step": x_ms,
                    "h2d_bytes_per_step": int(n * 32), "d2h_bytes_per_step": int(total + 24)},
            "gpu_launches": enc_launches * args.steps, "clocks": clocks.summary()}
    if not args.no_cpu_baseline:
        from oracle import ec_oracle as eco
        eco.build()
        m = min(n, 2_000_000)
        # whole planes only: cut at the first cluster of a plane
        key = cl_host["sector"][:m].astype(np.int64) * 256 + cl_host["row"][:m]
        m = int(np.searchsorted(key, key[-1])) if m < n else m
        t0 = time.perf_counter()
        buf, err, tot = eco.encode(cl_host[:m], geom[0], geom[1])
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": m / dt, "unit": "clusters/s", "cores": 1, "kind": "oracle",
                                "sample": "first %d clusters (whole planes) of the stream, %.1f s, single thread" % (m, dt)}
    print(json.dumps(line))
    coder.close()
    return 0


def run_shard(args):
    """--shard: one frame over the N ranks (paper_2402_01205_b200/shard.py).  A step = every rank's tpc_cf_run on its
    plane range + the variable-size gather of the clusters into rank 0; time = max over ranks; value = the frame's
    digits / that time (strong scaling: the total work is fixed)."""
    import torch
    import torch.distributed as dist
    from datagen import gen
    import paper_2402_01205_b200 as cf
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = "cuda:%d" % local_rank
    if not dist.is_initialized():
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", str(29400 + os.getpid() % 500))
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device(dev))
    cfg = gen.CONFIGS[args.config]
    geom = gen.geometry(args.config)
    digits = gen.generate(args.config)                                  # every rank generates the same frame
    part = cf.plane_partition(cf.plane_counts(digits, geom[0], geom[1]), world)[rank]
    mine = digits[part[2]:part[3]]
    n = int(mine.shape[0])
    finder = cf.ClusterFinder(*geom[:4], npads=geom[4], max_digits=max(n, 1), max_clusters=n // 10 + 1024, device=dev)
    d = cf.to_device(mine, device=dev)
    n_cl = [0]

    def step():
        finder.run(d, n, flags=cf.DIGITS_SORTED)
        st = finder.status.cpu().numpy().view(cf.STATUS)[0]              # the count decides the transfer size
        n_cl[0] = int(st["n_clusters"])
        return cf.gather_records(finder.clusters, n_cl[0], 32, 0)

    sampler = ClockSampler(local_rank).start()
    for _ in range(args.warmup):
        out, counts = step()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier()
    torch.cuda.synchronize()
    with sampler as clocks:
        ev0.record()
        for _ in range(args.steps):
            out, counts = step()
        ev1.record()
        torch.cuda.synchronize()
    dist.barrier()
    t = torch.tensor([ev0.elapsed_time(ev1)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item()) / args.steps
    if rank == 0:
        nd = int(digits.shape[0])
        peak, peak_src = load_peaks()
        line = {"metric": METRIC, "value": nd / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "u16/i32/f32", "data": "synthetic",
                "config": {"workload": "config%d: %s" % (args.config, cfg["label"]), "mode": "shard (one frame over the "
                           "ranks, contiguous plane ranges balanced by digits, clusters gathered into rank 0)",
                           "digits_per_frame": nd, "clusters_per_frame": int(sum(counts)),
                           "clusters_per_rank": counts, "rank0_planes": list(part[:2]),
                           "l2": "inputs larger than the 126 MB L2; no flush", "parallelism": "shard x%d" % world},
                "clusters_per_s": sum(counts) / (ms * 1e-3),
                "f_io": {"value": (8.0 * nd + 32.0 * sum(counts)) / (ms * 1e-3) / 1e9 / (peak * world),
                         "note": "compulsory I/O / time / (peak x ranks)"},
                "roofline": None, "cpu_baseline": None, "e2e": None,
                "gpu_launches": finder.last_launch_count() * args.steps, "clocks": clocks.summary()}
        print(json.dumps(line))
    finder.close()
    dist.destroy_process_group()
    return 0


def run_chain(args):
    """--stage chain: the paper's synchronous TPC chain around the cluster finder on one GPU, without a
    host round trip: raw samples -> tpc_fe_run -> digits -> tpc_cf_run -> clusters -> tpc_ec_encode -> container.  A step
    = one frame through all three calls; the digit and cluster counts that size the next call's arguments are read from
    the device status blocks (one small synchronising read each, inside the timed region)."""
    import torch
    from datagen import gen, fe_gen
    import paper_2402_01205_b200 as cf
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    dev = "cuda:0"
    torch.cuda.set_device(0)
    cfg = dict(gen.CONFIGS[args.config])
    if args.fe_sectors:
        cfg["n_sectors"] = min(cfg["n_sectors"], args.fe_sectors)
    ns, nr, mp, nt, npads = gen.geometry(cfg)
    W = cf.tpc_fe_pad_stride(mp)
    n_planes = ns * nr
    host_raw = np.empty((n_planes, nt, W), dtype=np.uint16)
    host_ped = np.empty((n_planes, W), dtype=np.uint16)
    n_truth = 0
    for s_ in range(ns):
        d = gen.generate(cfg, sectors=(s_, s_ + 1))
        n_truth += int(d.shape[0])
        fe_gen.raw_from_digits(d, ns, nr, mp, nt, npads=npads, seed=cfg["seed"], planes=(s_ * nr, (s_ + 1) * nr),
                               out=(host_raw[s_ * nr:(s_ + 1) * nr], host_ped[s_ * nr:(s_ + 1) * nr]))
    raw = torch.from_numpy(host_raw.view(np.int16)).to(dev)
    ped = torch.from_numpy(host_ped.view(np.int16)).to(dev)
    del host_raw
    pads = int(np.sum(npads)) if npads is not None else nr * mp
    cells = ns * pads * nt
    max_d = int(1.3 * n_truth) + 4096
    max_c = max_d // 8 + 1024
    flt = cf.FrontEndFilter(ns, nr, mp, nt, npads=npads, device=dev,
                            max_digits_per_plane=int(min((nt + 32) * W, max(8192, 2.0 * n_truth / n_planes + 64 * W))))
    finder = cf.ClusterFinder(ns, nr, mp, nt, npads=npads, max_digits=max_d, max_clusters=max_c, device=dev)
    coder = cf.ClusterCoder(ns, nr, max_c, device=dev)
    digits = torch.empty(max_d * 8, dtype=torch.uint8, device=dev)
    box = torch.empty(coder.max_encoded_bytes(max_c), dtype=torch.uint8, device=dev)
    res = {}

    def step():
        flt.run(raw, ped, digits, capacity=max_d, zs_threshold=3)
        fs = flt.read_status()
        finder.run(digits, fs["n_digits"], flags=cf.DIGITS_SORTED)
        st = finder.status.cpu().numpy().view(cf.STATUS)[0]
        coder.encode(finder.clusters, int(st["n_clusters"]), box)
        res.update(fe=fs, path=int(st["path"]), n_clusters=int(st["n_clusters"]), cf_overflow=int(st["overflow"]))

    sampler = ClockSampler(0).start()
    for _ in range(args.warmup):
        step()
    es = coder.read_status()
    if res["fe"]["overflow"] or res["path"] != 3 or res["cf_overflow"] or es["error"]:
        raise RuntimeError("chain run invalid: %r %r" % (res, es))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    with sampler as clocks:
        ev0.record()
        for _ in range(args.steps):
            step()
        ev1.record()
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    es = coder.read_status()
    launches = flt.last_launch_count() + finder.last_launch_count() + coder.last_launch_count()
    line = {"metric": "tpc_raw_samples_per_second_through_filter_finder_coder", "value": cells / (ms * 1e-3),
            "unit": "samples/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u16/i32/f32", "data": "synthetic",
            "config": {"workload": "filter -> cluster finder -> entropy coder on config%d: %s" % (args.config, cfg["label"]),
                       "stage": "chain", "sectors": ns, "valid_samples": cells, "raw_bytes": int(raw.numel() * 2),
                       "digits": res["fe"]["n_digits"], "clusters": res["n_clusters"], "container_bytes": es["bytes"],
                       "raw_to_container_ratio": raw.numel() * 2.0 / max(1, es["bytes"]),
                       "l2": "input (%.2f GB) larger than the 126 MB L2; no flush" % (raw.numel() * 2 / 1e9)},
            "frames_per_s": 1e3 / ms, "roofline": None, "cpu_baseline": None, "e2e": None,
            "gpu_launches": launches * args.steps, "clocks": clocks.summary()}
    print(json.dumps(line))
    flt.close(); finder.close(); coder.close()
    return 0


def run_fe(args):
    """--stage fe: the front-end filter (include/tpc_fe.h) on the raw samples of one frame of the chosen config
    (datagen/fe_gen.py's forward model over the config's digits).  One GPU.  A step = one tpc_fe_run (all its kernels)
    over the whole frame, resident in HBM; value = raw samples per second."""
    import torch
    from datagen import gen, fe_gen
    import paper_2402_01205_b200 as cf
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    dev = "cuda:0"
    torch.cuda.set_device(0)
    cfg = dict(gen.CONFIGS[args.config])
    if args.fe_sectors:
        cfg["n_sectors"] = min(cfg["n_sectors"], args.fe_sectors)
    ns, nr, mp, nt, npads = gen.geometry(cfg)
    W = cf.tpc_fe_pad_stride(mp)
    n_planes = ns * nr
    zs = 3
    t0 = time.perf_counter()
    host_raw = torch.empty((n_planes, nt, W), dtype=torch.int16, pin_memory=True)
    host_ped = torch.empty((n_planes, W), dtype=torch.int16, pin_memory=True)
    raw_np, ped_np = host_raw.numpy().view(np.uint16), host_ped.numpy().view(np.uint16)
    n_truth = 0
    for s in range(ns):
        d = gen.generate(cfg, sectors=(s, s + 1))
        n_truth += int(d.shape[0])
        fe_gen.raw_from_digits(d, ns, nr, mp, nt, npads=npads, seed=cfg["seed"], planes=(s * nr, (s + 1) * nr),
                               out=(raw_np[s * nr:(s + 1) * nr], ped_np[s * nr:(s + 1) * nr]))
    gen_s = time.perf_counter() - t0
    raw = host_raw.to(dev)
    ped = host_ped.to(dev)
    pads = int(np.sum(npads)) if npads is not None else nr * mp
    cells = ns * pads * nt                                     # valid samples
    cap_plane = int(min((nt + 32) * W, max(8192, 2.0 * n_truth / n_planes + 64 * W)))
    flt = cf.FrontEndFilter(ns, nr, mp, nt, npads=npads, max_digits_per_plane=cap_plane, device=dev)
    cap = int(1.3 * n_truth) + 4096
    out = torch.empty(cap * 8, dtype=torch.uint8, device=dev)
    step = lambda: flt.run(raw, ped, out, capacity=cap, zs_threshold=zs)
    sampler = ClockSampler(0).start()
    for _ in range(args.warmup):
        step()
    st = flt.read_status()
    if st["overflow"]:
        raise RuntimeError("bench run invalid: status %r" % (st,))
    n_dig = st["n_digits"]
    flt.set_profiling(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kern = []
    torch.cuda.synchronize()
    with sampler as clocks:
        ev0.record()
        for _ in range(args.steps):
            step()
        ev1.record()
        torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    for _ in range(min(args.steps, 5)):                       # the dominant kernel alone, by its own event pair
        step()
        kern.append(flt.profile_ms())
    flt.set_profiling(False)
    k_ms = float(np.mean(kern))
    peak, peak_src = load_peaks()
    # algorithmic bytes of k_fe_filter per launch: 2 B per valid sample read once, 8 B per kept sample staged,
    # pedestals and line counts
    alg = 2.0 * cells + 8.0 * n_dig + 2.0 * n_planes * W + 4.0 * n_planes * W
    # e2e: host raw (pinned) -> device, filter, digits and status back
    host_out = torch.empty(cap * 8, dtype=torch.uint8, pin_memory=True)
    e2e = None
    if not args.no_e2e:
        def e2e_step():
            raw.copy_(host_raw, non_blocking=True)
            ped.copy_(host_ped, non_blocking=True)
            step()
            s2 = flt.read_status()
            host_out[:s2["n_digits"] * 8].copy_(out[:s2["n_digits"] * 8], non_blocking=True)
            torch.cuda.synchronize()
        e2e_step()
        t0 = time.perf_counter()
        for _ in range(2):
            e2e_step()
        x_ms = (time.perf_counter() - t0) * 1e3 / 2
        e2e = {"value": cells / (x_ms * 1e-3), "unit": "samples/s", "ms_per_step": x_ms,
               "h2d_bytes_per_step": int(raw.numel() * 2 + ped.numel() * 2), "d2h_bytes_per_step": int(n_dig * 8 + 16)}
    line = {"metric": "tpc_raw_samples_filtered_per_second", "value": cells / (ms * 1e-3), "unit": "samples/s",
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u16/i32", "data": "synthetic",
            "config": {"workload": "front-end filter (TPC-FE v1) on the raw samples of config%d: %s" % (
                           args.config, cfg["label"]), "stage": "fe", "sectors": ns, "planes": n_planes,
                       "valid_samples": cells, "raw_bytes": int(raw.numel() * 2), "digits_out": n_dig,
                       "digits_of_the_generator": n_truth, "zs_threshold": zs, "gen_seconds": gen_s,
                       "l2": "input (%.2f GB) larger than the 126 MB L2; no flush" % (raw.numel() * 2 / 1e9)},
            "digits_per_s": n_dig / (ms * 1e-3),
            "roofline": {"bound": "hbm", "kernel": "k_fe_filter", "achieved": alg / (k_ms * 1e-3) / 1e9, "peak": peak,
                         "unit": "GB/s", "peak_source": peak_src, "frac": alg / (k_ms * 1e-3) / 1e9 / peak,
                         "traffic": load_traffic("config%d" % args.config, "fe", "k_fe_filter"),
                         "algorithmic_bytes_per_launch": alg, "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms},
            "cpu_baseline": None, "e2e": e2e, "gpu_launches": flt.last_launch_count() * args.steps,
            "clocks": clocks.summary()}
    if not args.no_cpu_baseline:
        from oracle import fe_oracle as feo
        feo.build()
        sp = min(n_planes, 3 * nr)
        t0 = time.perf_counter()
        od, ost = feo.run(raw_np[:sp], ped_np[:sp], max(1, sp // nr), nr, mp, nt, npads=npads, planes=(0, sp),
                          zs_threshold=zs)
        dt = time.perf_counter() - t0
        got = out[:ost["n_digits"] * 8].cpu().numpy()
        if got.tobytes() != od.tobytes():
            raise RuntimeError("bench: the filter's digits differ from the oracle's on the sample")
        sc = cells * sp / n_planes if npads is None else int(np.sum(npads)) * nt * (sp // nr)
        line["cpu_baseline"] = {"value": sc / dt, "unit": "samples/s", "cores": 1, "kind": "oracle",
                                "sample": "first %d planes (%d samples, %d digits, equal to the GPU's), %.1f s, "
                                          "single thread" % (sp, sc, ost["n_digits"], dt)}
    print(json.dumps(line))
    flt.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--path", default="fused", choices=["fused", "general"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--shuffle", action="store_true",
                    help="a seeded random permutation of the frame's digits, without the DIGITS_SORTED promise (the any-order "
                         "contract): digit sort on the device + fused path by default, the general path with --path "
                         "general; implies --no-e2e --no-per-config")
    ap.add_argument("--no-parity", action="store_true",
                    help="skip the element-by-element comparison of every cluster with the oracle (all host cores)")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false",
                    help="only the headline config (default: the other four configs of BASELINE.json are measured and "
                         "compared with the oracle too, in a per_config block of the same JSON line)")
    ap.add_argument("--variant", default="none", choices=["none", "flags", "cuts", "share"],
                    help="cluster-finder variants (SURVEY.md §8(f) NEXT #1): 'flags' = per-cluster flags, 'cuts' = "
                         "flags + q_tot_min 40 + single-pad cut, 'share' = flags + charge sharing between overlapping "
                         "clusters (V4, the K6 post-pass); the default run has none")
    ap.add_argument("--stage", default="cf", choices=["cf", "ec", "fe", "chain"],
                    help="'cf' = the cluster finder (the headline path); 'ec' = the entropy coder of the cluster stream "
                         "(SURVEY.md §8(f) NEXT #2): encode and decode of the frame's clusters, one JSON line; 'fe' = the "
                         "front-end filter (NEXT #3) on the frame's raw samples; 'chain' = filter -> cluster finder -> coder on "
                         "the device, one frame per step")
    ap.add_argument("--shard", action="store_true",
                    help="latency mode (SURVEY.md §8(e), NEXT #4): ONE frame is cut into contiguous plane ranges over the "
                         "N ranks, every rank runs the single-GPU path on its slice, rank 0 gathers the clusters "
                         "(scaling: strong)")
    ap.add_argument("--fe-sectors", type=int, default=0,
                    help="--stage fe: sectors of the frame to filter (0 = all of the config's)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.shuffle:
        args.no_e2e, args.per_config = True, False
    if args.impl == "reference":
        return run_reference(args)
    if args.stage == "ec":
        return run_ec(args)
    if args.stage == "fe":
        return run_fe(args)
    if args.stage == "chain":
        return run_chain(args)
    if args.shard:
        return run_shard(args)

    return run_cf(args)


# ---- comparison with the oracle (the bar of tests/parity.py, restated: bench.py does not import the tests) -------------
INT_FIELDS = ("sector", "row", "pad", "flags", "time", "qmax", "qtot", "rsv")
FLOAT_FIELDS = ("pad_mean", "time_mean", "sigma_pad", "sigma_time")


def compare_clusters(gpu, ora):
    """Element by element: integer fields bit-exact; floats pass iff |g-o| <= 1e-4 or <= 1e-5 |o| (north_star).
    Returns a dict for the JSON line; "ok" False on any mismatch."""
    res = {"clusters_gpu": int(gpu.shape[0]), "clusters_oracle": int(ora.shape[0]), "ok": True, "mismatch": None}
    if gpu.shape[0] != ora.shape[0]:
        res.update(ok=False, mismatch="cluster count")
        return res
    for f in INT_FIELDS:
        bad = int(np.count_nonzero(gpu[f] != ora[f]))
        if bad:
            res.update(ok=False, mismatch="%s differs at %d clusters" % (f, bad))
            return res
    err = {}
    for f in FLOAT_FIELDS:
        g, o = gpu[f].astype(np.float64), ora[f].astype(np.float64)
        e = np.abs(g - o)
        bad = int(np.count_nonzero(~((e <= 1e-4) | (e <= 1e-5 * np.abs(o)))))
        err[f] = float(e.max()) if e.size else 0.0
        if bad:
            res.update(ok=False, mismatch="%s out of tolerance at %d clusters" % (f, bad))
    res["max_abs_err"] = err
    res["clusters_checked"] = int(gpu.shape[0])
    return res


def measure_config(cf, torch, cfg_id, steps, warmup, path, variant, dev, frame_offset=0, parity=True, sampler=None,
                   keep=False, shuffle=False):
    """One config, device-resident: generate its frame(s), run `steps` timed steps (a step = every frame of the config
    through tpc_cf_run, back to back on one stream), time the dominant kernel by its own event pair, and compare every
    cluster of every frame with the oracle run on all host cores.  Returns a dict (and, with keep, the live objects)."""
    from datagen import gen
    cfg = gen.CONFIGS[cfg_id]
    geom = gen.geometry(cfg_id)
    n_frames = cfg["frames"]
    t0 = time.perf_counter()
    frames = [gen.generate(cfg_id, frame=frame_offset + f) for f in range(n_frames)]
    gen_s = time.perf_counter() - t0
    n_digits = [int(f.shape[0]) for f in frames]
    nmax = max(n_digits)
    max_clusters = nmax // 10 + 1024
    vflags = {"none": 0, "flags": cf.CLUSTER_FLAGS, "cuts": cf.CLUSTER_FLAGS | cf.CUT_SINGLE_PAD,
              "share": cf.CLUSTER_FLAGS | cf.SHARE_CHARGE}[variant]
    q_tot_min, q_saturation = (40 if variant == "cuts" else 0), (1000 if variant in ("flags", "cuts") else 0)
    finder = cf.ClusterFinder(*geom[:4], npads=geom[4], max_digits=nmax, max_clusters=max_clusters, device=dev,
                              q_tot_min=q_tot_min, q_saturation=q_saturation)
    flags = (cf.DIGITS_SORTED if path == "fused" else (cf.DIGITS_SORTED | cf.FORCE_GENERAL)) | vflags
    pinned = [torch.from_numpy(f.view(np.uint8)).pin_memory() for f in frames] if keep else None
    dev_digits = [(p if p is not None else torch.from_numpy(f.view(np.uint8))).to(dev, non_blocking=True)
                  for p, f in zip(pinned or [None] * n_frames, frames)]
    if shuffle:
        # any-order contract: a seeded random permutation of the device-resident digits, no
        # DIGITS_SORTED promise; the result must be the same array (R12), so the oracle still runs on the sorted frame
        gsh = torch.Generator(device=dev)
        gsh.manual_seed(2402)
        dev_digits = [d.view(torch.int64)[torch.randperm(n, device=dev, generator=gsh)].contiguous().view(torch.uint8)
                      for d, n in zip(dev_digits, n_digits)]
        flags = vflags | (cf.FORCE_GENERAL if path == "general" else 0)
    outs = [torch.empty(max_clusters * 32, dtype=torch.uint8, device=dev) for _ in frames]
    stats = [torch.zeros(32, dtype=torch.uint8, device=dev) for _ in frames]
    torch.cuda.synchronize()

    def step():
        for d, n, o, s in zip(dev_digits, n_digits, outs, stats):
            finder.run(d, n, flags=flags, clusters=o, status=s)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    sts = [finder.result(clusters=o, status=s)[1] for o, s in zip(outs, stats)]
    for st in sts:
        if st["path"] == 0 or st["overflow"]:
            raise RuntimeError("bench run invalid: status %r" % (st,))
    n_clusters = [st["n_clusters"] for st in sts]
    # inputs + outputs of one step against the 126 MB L2: small configs are timed with an L2 flush before every step
    step_bytes = 8 * sum(n_digits) + 32 * sum(n_clusters)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if step_bytes < (252 << 20) else None
    res = {"frames_per_step": n_frames, "digits": n_digits, "clusters": n_clusters,
           "launches_per_step": finder.last_launch_count() * n_frames, "kernel": finder.last_kernel(),
           "gen_seconds": gen_s, "occupancy": gen.occupancy(frames[0], cfg_id),
           "l2": ("inputs (%.2f GB digits per frame) larger than the 126 MB L2; no flush" % (nmax * 8 / 1e9)) if flush is None
                 else "step data (%.1f MB) fits the 126 MB L2: 256 MB written before every timed step (L2 flush)" % (step_bytes / 1e6)}
    finder.set_profiling(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ctx = sampler if sampler is not None else _NullCtx()
    with ctx:
        if flush is None:
            ev0.record()
            for _ in range(steps):
                step()
            ev1.record()
            torch.cuda.synchronize()
            total_ms = ev0.elapsed_time(ev1)
        else:
            total_ms = 0.0
            for _ in range(steps):
                flush.fill_(1)
                ev0.record()
                step()
                ev1.record()
                torch.cuda.synchronize()
                total_ms += ev0.elapsed_time(ev1)
    runs = steps * n_frames
    kern_ms = [finder.profile_ms(r, 1) for r in range(max(0, runs - 64), runs)]
    kern_ms = [k for k in kern_ms if k > 0]
    finder.set_profiling(False)
    res["total_ms"] = total_ms
    res["ms_per_step"] = total_ms / steps
    res["kernel_ms"] = float(np.mean(kern_ms)) if kern_ms else None
    del flush
    if parity:
        from oracle import oracle as orc
        orc.build()
        par = {"ok": True, "clusters_checked": 0, "frames": n_frames, "planes_per_frame": geom[0] * geom[1],
               "max_abs_err": {f: 0.0 for f in FLOAT_FIELDS}, "oracle": "all planes, all host cores"}
        t_or = 0.0
        for f, o, s in zip(frames, outs, stats):
            cl, st = finder.result(clusters=o, status=s)
            t0 = time.perf_counter()
            # (the variant bits have the same values on both sides: include/tpc_cf.h and oracle/tpc_cf_oracle.h)
            ora, ost, nthr = orc.run_parallel(f, *geom[:4], npads=geom[4], flags=vflags, q_tot_min=q_tot_min,
                                              q_saturation=q_saturation)
            t_or += time.perf_counter() - t0
            c = compare_clusters(cl, ora)
            if st["n_bad_digits"] != ost["n_bad_digits"]:
                c.update(ok=False, mismatch="n_bad_digits %d != %d" % (st["n_bad_digits"], ost["n_bad_digits"]))
            par["threads"] = nthr
            if not c["ok"]:
                par.update(ok=False, mismatch=c["mismatch"])
                break
            par["clusters_checked"] += c["clusters_checked"]
            for k, v in c["max_abs_err"].items():
                par["max_abs_err"][k] = max(par["max_abs_err"][k], v)
            del cl, ora
        par["oracle_seconds_all_cores"] = t_or
        res["parity"] = par
    if keep:
        res["_live"] = dict(finder=finder, frames=frames, pinned=pinned, dev_digits=dev_digits, outs=outs, stats=stats,
                            flags=flags, geom=geom, cfg=cfg, max_clusters=max_clusters)
    else:
        finder.close()
        del finder, dev_digits, outs, stats, frames
        torch.cuda.empty_cache()
    return res


class _NullCtx:
    def __enter__(self):
        return self

    def __exit__(self, *a):
        return False


def alg_bytes_of(path, nd, nc, geom):
    """Algorithmic bytes of one launch of the dominant kernel."""
    if path == "fused":
        # 8 B/digit read, 32 B/cluster staged, 4 B per pad line (peak count)
        return 8.0 * nd + 32.0 * nc + 4.0 * geom[0] * geom[1] * geom[2]
    # general: 8 B/digit read + the 3x3 neighbourhood of every digit >= threshold covered by the 2 B/digit map cells of
    # three lines (each map sector counted once) + 32 B/cluster staged + peak mask
    return 8.0 * nd + 2.0 * nd + 32.0 * nc + nd / 8.0


def run_cf(args):
    import torch
    import torch.distributed as dist
    from datagen import gen
    import paper_2402_01205_b200 as cf

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local_rank)
    dev = "cuda:%d" % local_rank
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    peak, peak_src = load_peaks()
    do_parity = not args.no_cpu_baseline and not args.no_parity and rank == 0

    # ---- headline config: K timed steps, device-resident inputs --------------------------------------------------------
    cfg = gen.CONFIGS[args.config]
    sampler = ClockSampler(local_rank).start()
    if world > 1:
        dist.barrier()
    # replicas: rank r works on its own frames (frame index offset by rank * frames)
    m = measure_config(cf, torch, args.config, args.steps, args.warmup, args.path, args.variant, dev,
                       frame_offset=rank * cfg["frames"], parity=do_parity, sampler=sampler, keep=True,
                       shuffle=args.shuffle)
    clocks = sampler
    live = m.pop("_live")
    finder, frames, pinned, dev_digits = live["finder"], live["frames"], live["pinned"], live["dev_digits"]
    geom, flags, max_clusters = live["geom"], live["flags"], live["max_clusters"]
    n_frames, n_digits, n_clusters = m["frames_per_step"], m["digits"], m["clusters"]
    if world > 1:
        dist.barrier()
    total_ms = m["total_ms"]
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        c = torch.tensor([sum(n_digits), sum(n_clusters)], dtype=torch.float64, device=dev)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
        digits_per_step, clusters_per_step = float(c[0].item()), float(c[1].item())
    else:
        digits_per_step, clusters_per_step = float(sum(n_digits)), float(sum(n_clusters))
    ms_per_step = total_ms / args.steps
    value = digits_per_step / (ms_per_step * 1e-3)

    # ---- e2e: the public call with HOST buffers (pinned), H2D + run + D2H of status and clusters, every step ----
    e2e = None
    if not args.no_e2e:
        host_out = torch.empty(max_clusters * 32, dtype=torch.uint8, pin_memory=True)
        e_steps = max(1, min(args.steps, 5))
        for p, d in zip(pinned, dev_digits):
            finder.run_host(p, flags=flags, dev_digits=d, host_clusters=host_out)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            for p, d in zip(pinned, dev_digits):
                cl, st = finder.run_host(p, flags=flags, dev_digits=d, host_clusters=host_out)
        torch.cuda.synchronize()
        e_ms = (time.perf_counter() - t0) * 1e3 / e_steps
        if world > 1:
            t = torch.tensor([e_ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e_ms = float(t.item())
        e2e = {"value": digits_per_step / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": e_ms,
               "h2d_bytes_per_step": int(sum(n_digits) * 8), "d2h_bytes_per_step": int(sum(n_clusters) * 32 + 32 * n_frames),
               "steps": e_steps}
        del host_out

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (HBM-bound: stencil/compaction work, no contraction) ----
    nd, nc = n_digits[-1], n_clusters[-1]     # per launch: one frame
    kname = m["kernel"]
    alg_bytes = alg_bytes_of(args.path, nd, nc, geom)
    k_ms = m["kernel_ms"]
    roof = {"bound": "hbm", "kernel": kname, "achieved": (alg_bytes / (k_ms * 1e-3) / 1e9) if k_ms else None,
            "peak": peak, "unit": "GB/s", "peak_source": peak_src,
            "frac": (alg_bytes / (k_ms * 1e-3) / 1e9 / peak) if k_ms else None,
            "traffic": load_traffic("config%d" % args.config, args.path, kname),
            "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": k_ms,
            "kernel_share_of_step": (k_ms * n_frames / ms_per_step) if k_ms else None}
    io_bytes = 8.0 * digits_per_step + 32.0 * clusters_per_step
    f_io = io_bytes / (ms_per_step * 1e-3) / 1e9 / peak

    # ---- the oracle on the host cores: one thread (the definition as it stands) and all cores (plane blocks) -------
    cpu = cpu_all = None
    if not args.no_cpu_baseline:
        from oracle import oracle as orc
        orc.build()
        ns = sample_sectors(args.config)
        hi = int(np.searchsorted(frames[0]["sector"], ns))
        sample = frames[0][:hi]
        dt, ost = time_oracle(sample, geom, ns)
        cpu = {"value": sample.shape[0] / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": "first %d of %d sectors of frame 0 (%d digits, %d clusters), %.1f s, single thread" % (
                   ns, geom[0], sample.shape[0], ost["n_clusters"], dt),
               "clusters_per_s": ost["n_clusters"] / dt, "host_cores_available": os.cpu_count()}
        if do_parity and m.get("parity"):
            t_all = m["parity"]["oracle_seconds_all_cores"] / n_frames
            cpu_all = {"value": n_digits[0] / t_all, "unit": UNIT, "cores": m["parity"].get("threads"), "kind": "oracle",
                       "sample": "frame 0, all %d planes, the single-threaded routine on plane blocks from %s host threads, "
                                 "%.1f s; its output is the array the GPU's clusters are compared with" % (
                                     geom[0] * geom[1], m["parity"].get("threads"), t_all),
                       "clusters_identical_to_single_thread": None}
            if ns == geom[0]:
                # the all-cores run must reproduce the single-threaded one: compare counts (the arrays themselves
                # were compared with the GPU's, which equals both if it equals one)
                cpu_all["clusters_identical_to_single_thread"] = bool(ost["n_clusters"] == n_clusters[0])

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u16/i32/f32", "data": "synthetic",
            "config": {"workload": "config%d: %s" % (args.config, cfg["label"]), "path": args.path,
                       "variant": args.variant, "digit_order": "shuffled (seeded permutation)" if args.shuffle else "sorted",
                       "frames_per_step": n_frames, "digits_per_frame": nd, "clusters_per_frame": nc,
                       "occupancy": m["occupancy"], "parallelism": "replicas x%d" % world,
                       "l2": m["l2"],
                       "checksum_frame0": "%016x" % gen.checksum(frames[0]) if nd < 50_000_000 else "skipped (large)",
                       "gen_seconds": m["gen_seconds"]},
            "clusters_per_s": clusters_per_step / (ms_per_step * 1e-3),
            "f_io": {"value": f_io, "bytes_per_step": io_bytes, "note": "compulsory I/O (8 B/digit + 32 B/cluster) / time / peak"},
            "roofline": roof, "cpu_baseline": cpu, "cpu_baseline_all_cores": cpu_all, "parity": m.get("parity"),
            "e2e": e2e, "gpu_launches": m["launches_per_step"] * args.steps, "clocks": clocks.summary()}
    finder.close()
    del finder, dev_digits, frames, pinned, live
    torch.cuda.empty_cache()

    # ---- every other config of BASELINE.json (north_star: "digits/s and clusters/s ... for each config") -------------
    ok = not (line["parity"] and not line["parity"]["ok"])
    if args.per_config and world == 1 and args.variant == "none":
        per = {}
        for c in (1, 2, 3, 4, 5):
            if c == args.config:
                continue
            try:
                r = measure_config(cf, torch, c, max(5, min(args.steps, 20)), args.warmup, args.path, "none", dev,
                                   parity=do_parity)
            except Exception as e:                      # e.g. not enough device or host memory for the 1.09e9-digit frame
                per["config%d" % c] = {"error": "%s: %s" % (type(e).__name__, e)}
                torch.cuda.empty_cache()
                continue
            g = gen.geometry(c)
            nd_c, nc_c = r["digits"][-1], r["clusters"][-1]
            ab = alg_bytes_of(args.path, nd_c, nc_c, g)
            ms = r["ms_per_step"]
            e = {"workload": "config%d: %s" % (c, gen.CONFIGS[c]["label"]), "frames_per_step": r["frames_per_step"],
                 "digits_per_frame": nd_c, "clusters_per_frame": nc_c, "ms_per_step": ms,
                 "ms_per_frame": ms / r["frames_per_step"], "digits_per_s": sum(r["digits"]) / (ms * 1e-3),
                 "clusters_per_s": sum(r["clusters"]) / (ms * 1e-3),
                 "f_io": (8.0 * sum(r["digits"]) + 32.0 * sum(r["clusters"])) / (ms * 1e-3) / 1e9 / peak,
                 "kernel": r["kernel"], "kernel_ms": r["kernel_ms"],
                 "roofline_frac": (ab / (r["kernel_ms"] * 1e-3) / 1e9 / peak) if r["kernel_ms"] else None,
                 "gpu_launches_per_step": r["launches_per_step"], "l2": r["l2"], "occupancy": r["occupancy"],
                 "parity": r.get("parity")}
            if r.get("parity"):
                t_all = r["parity"]["oracle_seconds_all_cores"]
                e["cpu_baseline_all_cores"] = {"value": sum(r["digits"]) / t_all, "unit": UNIT,
                                               "cores": r["parity"].get("threads"), "kind": "oracle"}
                ok = ok and r["parity"]["ok"]
            per["config%d" % c] = e
        line["per_config"] = per
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
