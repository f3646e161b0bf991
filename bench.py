#!/usr/bin/env python
"""bench.py — fused encode+MLP throughput of the OctaOctree query on B200 (BASELINE.json metric), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1|2|3|4] [--scaling weak|strong]
                  [--path auto|mma|tc|tm|unfused|generic]

A "step" is one pass of the whole hot path (a2-a9) over one frame of synthetic primary hits (config 1: 1024x1024).
`value` = queries/s with the queries already resident in HBM, timed per step with CUDA events on the launching stream,
L2 flushed between steps; `e2e` = the same through oo_query_host with pinned HOST buffers (H2D + kernel + D2H inside the
timed region).  N > 1: one process per GPU; from a plain shell (`python bench.py --gpus N`, no WORLD_SIZE in the
environment) the script re-launches itself under `python -m torch.distributed.run --nproc-per-node N`.  The cache is
replicated on every GPU (read-only); `--scaling weak` (default): every rank renders its OWN frame (camera seed = rank), no
data-path collective; `--scaling strong`: ONE frame is split into contiguous query slices (dist.shard_range), every rank
evaluates its slice and the RGB slices are all-gathered over NCCL inside the timed region, so every rank ends the step
holding the whole frame.  Timings are the max over ranks.  `--impl reference` times the CPU oracle (oracle/) as it stands.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fused encode+MLP query throughput"
UNIT = "Mqueries/s"


def workload_for(cfg: int, rank: int = 0):
    """The BASELINE.json workload of configs[cfg].  rank > 0 (weak scaling): the same scene, cache and decoder with that
    rank's own frame -- another seeded camera pose (configs 1-3) or another stretch of the incoherent sampler (config 4)."""
    import gen
    if cfg == 4:
        # BASELINE.json configs[4], the incoherent distribution at 2^22 queries: config 3's scene, tree, atlas and MLP; queries =
        # area-weighted surface samples in random order (the batch-size x distribution table is --sweep 4)
        w = gen.scene_workload(3, seed=0, width=64, height=64, incoherent_n=1 << 22)
        w.meta["width"], w.meta["height"], w.meta["incoherent"] = 2048, 2048, True   # width/height only cut the CPU oracle's sample into index ranges
        if rank:
            w.queries = gen.incoherent_queries(w.scene, 1 << 22, 0, first=rank << 22)
    else:
        w = gen.scene_workload(cfg, seed=0)
        if rank:
            w.camera = gen.make_camera(w.meta["width"], w.meta["height"], rank)
            ex = w.queries.extra
            w.queries = gen.raycast(w.scene, w.camera)
            if ex is not None:
                w.queries.extra = gen.roughness(w.queries.n, rank)
    L, F = len(w.tree.level_depth), w.atlas.F
    n_extra = 0 if w.queries.extra is None else w.queries.extra.shape[1]
    texel = F * 2
    gather = L * 4 * texel
    io = 36 + 4 * n_extra + 12
    dims = [w.mlp.in_dim] + [64] * w.mlp.n_hidden + [3]
    flops = 2 * sum(a * b for a, b in zip(dims[:-1], dims[1:]))
    desc = {
        "workload": "BASELINE.json configs[%d]: %s (%d queries, %s), adaptive octree depth %d "
                    "(%d nodes), used depths %s, R_l %s, F=%d fp16, MLP %d->%dx64->3 exp" %
                    (cfg, "incoherent queries on the config-3 cache: x area-weighted on the scene surfaces, wo uniform on the hemisphere" if cfg == 4
                     else "%dx%d primary-hit frame" % (w.meta["width"], w.meta["height"]), w.queries.n,
                     "random order" if cfg == 4 else "scanline order", w.tree.max_depth, w.tree.n_nodes,
                     w.tree.level_depth, w.tree.level_res, F, w.mlp.in_dim, w.mlp.n_hidden),
        "queries_per_step": w.queries.n, "bytes_per_query": gather + io, "gather_bytes_per_query": gather,
        "flop_per_query": flops, "atlas_bytes": w.atlas.nbytes,
    }
    return w, desc


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 1590.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1590.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons, sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows]
        sm = sorted(float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit())
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in rows for k in range(4) if len(r) > 2 + k and r[2 + k].lower().startswith("active")})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(rows)}


def oracle_sample(w, target_queries: int):
    """A bounded sample of the same frame for the CPU oracle: whole scanlines at a fixed row stride."""
    import numpy as np
    W, H = w.meta["width"], w.meta["height"]
    rows = max(1, min(H, target_queries // W))
    stride = max(1, H // rows)
    ridx = np.arange(0, H, stride)[:rows]
    idx = (ridx[:, None] * W + np.arange(W)[None, :]).ravel()
    if w.meta.get("incoherent"):
        return w.queries.take(idx), "%d queries = %d runs of %d consecutive queries (every %dth run) of the random-order batch" % (len(idx), len(ridx), W, stride)
    return w.queries.take(idx), "%d queries = %d scanlines (every %dth row) of the %dx%d frame" % (len(idx), len(ridx), stride, W, H)


def time_oracle(w, sample_q, repeats: int = 1):
    from oracle import c as OC
    co = OC.from_workload(w)
    co.query(sample_q.x[:1024], sample_q.nrm[:1024], sample_q.wo[:1024], None if sample_q.extra is None else sample_q.extra[:1024])
    best, threads = None, 1
    for _ in range(repeats):
        t0 = time.perf_counter()
        _, threads = co.query(sample_q.x, sample_q.nrm, sample_q.wo, sample_q.extra, return_threads=True)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best, threads


def run_reference(args):
    """The reference arm of this tier = the CPU oracle as it stands.  EXACTLY K timed steps after W warm-ups; a step is a
    bounded sample of the frame (whole scanlines at a fixed stride), sized from a short calibration so that W + K steps end
    within about --ref-budget seconds (the whole frame when it fits)."""
    rank, _, world = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("LOCAL_RANK", "0"), ("WORLD_SIZE", "1")))
    if rank != 0:
        return 0
    w, desc = workload_for(args.config)
    cal_q, _ = oracle_sample(w, 65536)
    dt_cal, _ = time_oracle(w, cal_q)
    rate = cal_q.n / dt_cal
    per_step = int(rate * args.ref_budget / max(1, args.steps + args.warmup))
    sample_q, sample_desc = oracle_sample(w, max(w.meta["width"], min(w.queries.n, per_step)))
    for _ in range(args.warmup):
        time_oracle(w, sample_q)
    times, threads = [], 1
    for _ in range(args.steps):
        dt, threads = time_oracle(w, sample_q)
        times.append(dt)
    mean = sum(times) / len(times)
    val = sample_q.n / mean / 1e6
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": mean * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": desc, "run": {"sample": sample_desc},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample_desc},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "note": "the CPU oracle (oracle/oo_oracle.c, double precision, OpenMP over queries) as it stands; each step = the bounded sample"}
    print(json.dumps(out))
    return 0


PATH_NAMES = {0: "auto", 1: "generic", 2: "unfused", 3: "fused_mma", 4: "fused_tcgen05", 5: "fused_tcgen05_tmem_a", 6: "full_query"}


def source_sha() -> str:
    """Hash of the CUDA sources the library is built from: stamps profiles/traffic.json so that a stale capture is refused."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_08469_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_facts(cfg: int):
    """Per-launch facts of the dominant kernel from the committed ncu capture (profiles/traffic.json): DRAM bytes and warp
    instructions.  Valid only for the sources they were captured from: a stamp mismatch returns (None, reason)."""
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(tp):
        return None, "no profiles/traffic.json"
    d = json.load(open(tp))
    e = d.get("cfg%d" % cfg)
    if not e:
        return None, "no capture for config %d" % cfg
    if e.get("source_sha") != source_sha():
        return None, "stale: captured from other kernel sources (%s, now %s); re-run the ncu pass and bench.py --ingest-ncu" % (e.get("source_sha"), source_sha())
    return e, None


def ingest_ncu(args):
    """bench.py --ingest-ncu CSV --config K: read an `ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum,
    smsp__inst_executed.sum,gpu__time_duration.sum --csv --log-file CSV python bench.py --quick --config K ...` launch list and
    store the last full-size launch of the dominant kernel (name contains --ingest-kernel, default 'fused') in profiles/traffic.json,
    stamped with the hash of the kernel sources."""
    import csv
    rows = [r for r in csv.reader(l for l in open(args.ingest_ncu) if l.startswith('"'))]
    head, rows = rows[0], rows[1:]
    k_id, k_name, k_metric, k_val = head.index("ID"), head.index("Kernel Name"), head.index("Metric Name"), head.index("Metric Value")
    launches = {}
    for r in rows:
        if args.ingest_kernel in r[k_name]:
            launches.setdefault(int(r[k_id]), {"kernel": r[k_name].split("(")[0]})[r[k_metric]] = float(r[k_val].replace(",", ""))
    if not launches:
        raise SystemExit("no launch of a kernel matching %r in %s" % (args.ingest_kernel, args.ingest_ncu))
    # the step's launch: among the launches with the most instructions (not the smaller ones of the e2e leg's chunks) the last one that
    # ran from device memory (the e2e leg's zero-copy launch executes the same instructions but reads its queries over PCIe and takes
    # many times longer)
    key = "smsp__inst_executed.sum" if any("smsp__inst_executed.sum" in v for v in launches.values()) else "gpu__time_duration.sum"
    top = max(v.get(key, 0) for v in launches.values())
    full = {i: v for i, v in launches.items() if v.get(key, 0) >= 0.99 * top}
    fastest = min(v.get("gpu__time_duration.sum", 0) for v in full.values())
    m = full[max(i for i, v in full.items() if v.get("gpu__time_duration.sum", 0) <= 1.5 * fastest)]
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    d = json.load(open(tp)) if os.path.exists(tp) else {}
    d.pop("source", None)
    d["how"] = ("per launch of the dominant kernel, --clock-control none: ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum,"
                "smsp__inst_executed.sum,gpu__time_duration.sum --csv --log-file X.csv python bench.py --quick --config K --steps 5 --warmup 3; "
                "python bench.py --ingest-ncu X.csv --config K")
    d["cfg%d" % args.config] = {"dram_bytes_per_launch": int(m.get("dram__bytes_read.sum", 0) + m.get("dram__bytes_write.sum", 0)),
                                "warp_instructions_per_launch": int(m.get("smsp__inst_executed.sum", 0)),
                                "ncu_time_ns": int(m.get("gpu__time_duration.sum", 0)), "kernel": m["kernel"], "source_sha": source_sha()}
    json.dump(d, open(tp, "w"), indent=1)
    print(json.dumps(d["cfg%d" % args.config]))
    return 0


def compulsory_bytes(ctx, w, x, nrm, wo, ex):
    """What one frame MUST read from DRAM if every distinct byte were fetched once: the distinct 32-byte sectors (and distinct
    texels) of the padded atlas the frame's taps touch, counted from the fused kernel's own indices (oo_query_debug), plus the
    query stream in and the RGB out.  The gap between this and L*4*texel bytes per query is the reuse neighbouring queries share."""
    import torch
    rgb, slot, tex = ctx.oo_query_debug(x, nrm, wo, ex)
    del rgb
    tb = w.atlas.F * 2
    uniq_texels = uniq_sectors = 0
    for l, R in enumerate(w.tree.level_res):
        Rp = R + 2
        s = slot[:, l].long()
        ok = s >= 0
        base = s[ok] * (Rp * Rp) + (tex[ok][:, l, 1].long() + 1) * Rp + (tex[ok][:, l, 0].long() + 1)      # padded texel index of tap (i0, j0)
        taps = torch.cat([base, base + 1, base + Rp, base + Rp + 1])
        ut = torch.unique(taps)
        uniq_texels += int(ut.numel())
        uniq_sectors += int(torch.unique((ut * tb) // 32).numel()) if tb < 32 else int(ut.numel()) * (tb // 32)
        del s, ok, base, taps, ut
    n, ne = int(x.shape[0]), 0 if ex is None else int(ex.shape[1])
    io = n * (36 + 4 * ne + 12)
    return {"distinct_texel_bytes": uniq_texels * tb, "distinct_sector_bytes": uniq_sectors * 32, "query_io_bytes": io,
            "total": uniq_sectors * 32 + io, "how": "distinct padded-atlas texels / 32-byte sectors touched by the frame's 4 taps per level (from oo_query_debug's indices) + 36 B in + 12 B out per query"}


def relaunch_if_needed(args) -> int:
    """`python bench.py --gpus N` from a plain shell: start N ranks (one per GPU) of this same command under torch.distributed.run.
    Returns the children's exit code, or -1 when this process is already a rank (or N == 1) and should carry on."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ:
        return -1
    import socket
    if not args.dry_run_dist:
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            sys.stderr.write("bench.py: --gpus %d but %d CUDA device(s) visible\n" % (args.gpus, have))
            return 2
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")               # NCCL's init log names every rank and the transport (NVLS / P2P) ...
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    env.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")   # ... on stderr: stdout stays the one JSON line
    env.setdefault("OMP_NUM_THREADS", str(max(1, (os.cpu_count() or 1) // args.gpus)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def run_dry_dist(args):
    """--dry-run-dist: the N > 1 host logic of the product arm with the gloo backend and no GPU -- launcher, rank environment,
    per-rank frames (weak) or shard_range slices + all_gather_rows (strong), max/sum reductions, one JSON line from rank 0.
    The per-query work is replaced by a stand-in (rgb = x), so this measures nothing: it is what the CPU tests drive."""
    import numpy as np
    import torch
    import gen
    from paper_2606_08469_b200 import dist as D
    rank, local_rank, world = D.env_rank_world()
    if world > 1:
        D.init_process_group("gloo")
    scene = gen.make_scene("three", 0)
    n_frame = 96 * 64
    if args.scaling == "strong":
        q = gen.raycast(scene, gen.make_camera(96, 64, 0))
        lo, hi = D.shard_range(q.n, rank, world)
        local = torch.from_numpy(q.x[lo:hi].copy())
        full = D.all_gather_rows(local, q.n)
        assert torch.equal(full, torch.from_numpy(q.x)), "all_gather_rows did not rebuild the frame"
        mine, checksum = hi - lo, float(full.double().sum())
    else:
        q = gen.raycast(scene, gen.make_camera(96, 64, rank))
        mine, checksum = q.n, float(torch.from_numpy(q.x).double().sum())
    (mx,), (tot, chk) = D.reduce_max_sum([1.0 + rank], [mine, checksum if args.scaling == "weak" else 0.0], torch.device("cpu"))
    if rank == 0:
        print(json.dumps({"dry_run": True, "n_gpus": world, "scaling": args.scaling, "queries": int(tot), "frame": n_frame,
                          "dist_ranks": torch.distributed.get_world_size() if world > 1 else None,
                          "max_ms": mx, "checksum": checksum if args.scaling == "strong" else chk}))
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import paper_2606_08469_b200 as P
    from paper_2606_08469_b200 import dist as D
    rank, local_rank, world = D.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        D.init_process_group("nccl")
    strong = args.scaling == "strong" and world > 1
    w, desc = workload_for(args.config, 0 if args.scaling == "strong" else rank)
    q = w.queries
    n_frame = q.n
    lo, hi = D.shard_range(q.n, rank, world) if strong else (0, q.n)
    ctx = P.OctaOctree(local_rank).upload_workload(w)
    path = {"auto": P.PATH_AUTO, "mma": P.PATH_FUSED_MMA, "tc": P.PATH_FUSED_TC, "tm": P.PATH_FUSED_TC_TMEM, "unfused": P.PATH_UNFUSED, "generic": P.PATH_GENERIC}[args.path]
    ctx.oo_set_path(path)
    ctx.oo_set_presort(args.presort)              # default "auto": what a caller who sets nothing gets
    ctx.oo_reserve(q.n)
    cu = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a[lo:hi])).to(dev)
    x, nrm, wo, ex = cu(q.x), cu(q.nrm), cu(q.wo), cu(q.extra)
    n_mine = hi - lo
    rgb = torch.empty((n_mine, 3), dtype=torch.float32, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)          # > 126 MB L2
    stream = torch.cuda.current_stream(dev)
    frame = [None]

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    def timed(n_steps, do_flush, fn):
        evs = []
        for _ in range(n_steps):
            if do_flush:
                flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            evs.append((e0, e1))
        torch.cuda.synchronize(dev)
        return [a.elapsed_time(b) for a, b in evs]

    encode_only = args.phase == "encode"
    feat = torch.empty((n_mine, len(w.tree.level_depth) * w.atlas.F), dtype=torch.float16, device=dev) if encode_only else None

    def step():
        if encode_only:   # the encoding phase alone (a2-a6): features round-trip HBM; side measurement, the ncu target of north_star's "encoding phase"
            ctx.oo_encode(x, wo, features=feat)
            return
        ctx.oo_query(x, nrm, wo, ex, rgb=rgb)
        if strong:        # the path's one optional exchange: every rank ends the step with the whole frame (NCCL all-gather)
            frame[0] = D.all_gather_rows(rgb, n_frame)

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = ctx.oo_get_info()["query_launches"]
    t0 = time.time()
    barrier()
    ms = timed(args.steps, True, step)
    barrier()
    t1 = time.time()
    launches = ctx.oo_get_info()["query_launches"] - l0
    # keep the GPU under the same load a little longer so that the 100 ms clock sampler sees it (not part of the number)
    if sampler and (t1 - t0) < 0.5 and not args.quick:
        tend = time.time() + 0.5
        while time.time() < tend:
            step() if encode_only else ctx.oo_query(x, nrm, wo, ex, rgb=rgb)
        torch.cuda.synchronize(dev)
        t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms_warm = timed(min(args.steps, 50), False, step) if not args.quick else ms
    if encode_only:
        mean_ms, warm_ms = sum(ms) / len(ms), sum(ms_warm) / len(ms_warm)
        hbm, tf, which = peaks()
        L, F = len(w.tree.level_depth), w.atlas.F
        bq = desc["gather_bytes_per_query"] + 24 + L * F * 2        # x, wo in; fp16 feature row out
        info = ctx.oo_get_info()
        print(json.dumps({"metric": "encode-only query throughput (a2-a6, features to HBM)", "value": n_mine / (mean_ms * 1e-3) / 1e6, "unit": UNIT,
                          "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": mean_ms, "ms_per_step_warm_l2": warm_ms,
                          "config": desc, "run": {"presort": args.presort, "presorted": bool(info["presorted_last_encode"]), "l2": "flushed between steps",
                                                  "path": PATH_NAMES[info["path_last_encode"]]},
                          "clocks": clocks, "gpu_launches": int(launches), "dtype": "f16", "data": "synthetic",
                          "roofline": {"bound": "hbm", "achieved": bq * n_mine / (mean_ms * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                                       "frac": bq * n_mine / (mean_ms * 1e-3) / 1e9 / hbm, "bytes_per_query": bq, "peak_source": which}}))
        return 0
    checksum_dev = float((frame[0] if strong else rgb).double().sum())
    strong_ok = None
    if strong:
        # outside the timed region: every rank evaluates the WHOLE frame alone (the cache is replicated) and compares it with the frame the
        # all-gather assembled.  RGB per query does not depend on the sharding, so the two are equal bit for bit; a run where they are not
        # fails on every rank at once (no rank is left waiting in a collective).
        cuf = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        alone = ctx.oo_query(cuf(q.x), cuf(q.nrm), cuf(q.wo), cuf(q.extra))
        torch.cuda.synchronize(dev)
        strong_ok = bool(torch.equal(alone, frame[0]))
        if not strong_ok:
            raise SystemExit("bench.py: rank %d: the all-gathered frame differs from the same frame evaluated on one rank "
                             "(checksums %r vs %r)" % (rank, checksum_dev, float(alone.double().sum())))
        del alone
    # e2e: pinned host buffers, H2D + kernels + D2H inside the timed region, through oo_query_host
    pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a[lo:hi])).pin_memory()
    hx, hn, hw, he = pin(q.x), pin(q.nrm), pin(q.wo), pin(q.extra)
    hrgb = torch.empty((n_mine, 3), dtype=torch.float32).pin_memory()
    e2e_steps = max(3, min(args.steps, 20)) if not args.quick else 1
    for _ in range(0 if args.quick else 2):
        ctx.oo_query_host(hx, hn, hw, he, rgb=hrgb)
    barrier()
    e2e_times = []
    for _ in range(e2e_steps):
        te = time.perf_counter()
        ctx.oo_query_host(hx, hn, hw, he, rgb=hrgb)          # synchronous: returns when the RGB is in host memory
        e2e_times.append((time.perf_counter() - te) * 1e3)
    torch.cuda.synchronize(dev)
    e2e_ms = sum(e2e_times) / len(e2e_times)
    checksum = float(hrgb.double().sum())
    e2e_zero_copy = bool(ctx.oo_get_info()["host_zero_copy_last"])
    pipeline_ms = None
    if e2e_zero_copy and not args.quick:           # for comparison: the same call through the chunked copy pipeline
        ctx.oo_set_host_zero_copy(False)
        ctx.oo_query_host(hx, hn, hw, he, rgb=hrgb)
        tt = []
        for _ in range(5):
            te = time.perf_counter()
            ctx.oo_query_host(hx, hn, hw, he, rgb=hrgb)
            tt.append((time.perf_counter() - te) * 1e3)
        pipeline_ms = sum(tt) / len(tt)
        ctx.oo_set_host_zero_copy(True)
    # measured copy rates of this box (one 64 MB pinned copy each way), so that the PCIe floor of e2e is a measured number
    h2d_gbs = d2h_gbs = None
    if not args.quick and rank == 0:
        hb, db = torch.empty(64 << 20, dtype=torch.uint8).pin_memory(), torch.empty(64 << 20, dtype=torch.uint8, device=dev)
        for direction in (0, 1):
            best = 1e9
            for _ in range(5):
                torch.cuda.synchronize(dev)
                tc = time.perf_counter()
                (db.copy_(hb, non_blocking=True) if direction == 0 else hb.copy_(db, non_blocking=True))
                torch.cuda.synchronize(dev)
                best = min(best, time.perf_counter() - tc)
            if direction == 0:
                h2d_gbs = (64 << 20) / best / 1e9
            else:
                d2h_gbs = (64 << 20) / best / 1e9

    mean_ms, warm_ms = sum(ms) / len(ms), sum(ms_warm) / len(ms_warm)
    (mx_ms, mx_warm, mx_e2e), (tot_q, chk_sum) = D.reduce_max_sum([mean_ms, warm_ms, e2e_ms], [n_mine, checksum], dev)
    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return 0
    hbm, tf, which = peaks()
    value = tot_q / (mx_ms * 1e-3) / 1e6
    ne = 0 if q.extra is None else q.extra.shape[1]
    alg_bytes = desc["bytes_per_query"] * n_mine                 # rank 0's launch (every rank's is the same size +- 1 query)
    achieved = alg_bytes / (mean_ms * 1e-3) / 1e9
    flop_time = desc["flop_per_query"] * n_mine / (tf * 1e12)
    byte_time = alg_bytes / (hbm * 1e9)
    info = ctx.oo_get_info()
    facts, stale = (None, "not looked up") if strong else ncu_facts(args.config)
    roof = {"bound": "hbm", "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm,
            "traffic": facts["dram_bytes_per_launch"] if facts else None,
            "peak_source": which, "kernel": "fused encode+MLP (one launch per step)" if not info["presorted_last_query"] else
            "whole step: histogram + scan + bin_scatter + fused encode+MLP on the binned copy + unbin (traffic is the fused launch's)",
            "definition": "BASELINE.json north_star: ALGORITHMIC bytes (L*4 texels gathered + 36 B in + 12 B out per query) at the measured HBM peak, "
                          "vs the MLP FLOPs at the dense fp16 peak; the slower of the two is the roofline",
            "roofline_ms": max(byte_time, flop_time) * 1e3, "flop_time_ms": flop_time * 1e3, "byte_time_ms": byte_time * 1e3,
            "binds": "bytes" if byte_time >= flop_time else "flops",
            "frac_warm_l2": alg_bytes / (warm_ms * 1e-3) / 1e9 / hbm}
    if roof["frac"] > 1.0:
        roof["frac_note"] = ("above 1: neighbouring queries share texels, so L1/L2 serve bytes the algorithmic count charges to HBM; for this "
                             "config the algorithmic-byte figure is not a bound -- see dram / compulsory / issue below")
    if facts:
        dram = facts["dram_bytes_per_launch"]
        roof["dram"] = {"bytes_per_launch": dram, "GBps": dram / (mean_ms * 1e-3) / 1e9, "frac_of_peak": dram / (mean_ms * 1e-3) / 1e9 / hbm,
                        "vs_algorithmic": dram / alg_bytes, "kernel": facts.get("kernel"), "source": "profiles/traffic.json (ncu, stamped %s)" % facts["source_sha"]}
        wi = facts.get("warp_instructions_per_launch")
        if wi and clocks and clocks.get("sm_mhz"):
            # second bound: every warp instruction needs one issue slot; an SM issues 4 per cycle (one per sub-partition)
            issue_ms = wi / (info["n_sms"] * 4 * clocks["sm_mhz"] * 1e6) * 1e3
            roof["issue"] = {"warp_instructions_per_launch": wi, "thread_instructions_per_query": wi * 32 / n_mine, "bound_ms": issue_ms,
                             "frac": issue_ms / mean_ms, "how": "warp instructions / (SMs x 4 issue slots x measured SM clock): the time below which this "
                             "instruction stream cannot run; frac = share of issue slots used"}
    else:
        roof["traffic_note"] = stale
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": mx_ms, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None, "dtype": "f16",
        "data": "synthetic", "config": desc,
        "run": {"l2": "flushed between steps (256 MB memset)", "path": PATH_NAMES[info["path_last_query"]], "ms_per_frame_warm_l2": mx_warm,
                "presort": args.presort, "presorted": bool(info["presorted_last_query"]), "coherence_distinct_cells_per_32_queries": info["coherence_x100"] / 100.0,
                "queries_per_rank": n_mine, "checksum_device": checksum_dev, "strong_checksum_matches_one_rank": strong_ok,
                "nccl_ranks": torch.distributed.get_world_size() if world > 1 else None,
                "parallelism": ("one GPU" if world == 1 else
                                "replicated cache; ONE frame split into contiguous query slices, RGB all-gathered over NCCL inside the timed region" if strong else
                                "replicated cache; every rank its own frame (camera seed = rank); no data-path collective")},
        "clocks": clocks,
        "e2e": {"value": tot_q / (mx_e2e * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": int((36 + 4 * ne) * n_mine),
                "d2h_bytes_per_step": int(12 * n_mine), "ms_per_step": mx_e2e, "ms_min": min(e2e_times), "ms_max": max(e2e_times),
                "api": "oo_query_host (pinned host buffers)" + (": one launch reads the queries from host memory in place and writes the RGB back (zero-copy)" if e2e_zero_copy
                                                                  else ": chunked copy-in / kernel / copy-out pipeline"),
                "copy_pipeline_ms": pipeline_ms, "checksum": chk_sum if not strong else checksum,
                "h2d_GBps_measured": h2d_gbs, "d2h_GBps_measured": d2h_gbs,
                "pcie_floor_ms": None if not h2d_gbs else (36 + 4 * ne) * n_mine / (h2d_gbs * 1e9) * 1e3},
        "gpu_launches": int(launches),
        "roofline": roof,
    }
    if world == 1 and not args.quick:
        try:
            roof["compulsory"] = comp = compulsory_bytes(ctx, w, x, nrm, wo, ex)
            roof["compulsory"]["byte_time_ms"] = comp["total"] / (hbm * 1e9) * 1e3
            roof["compulsory"]["frac"] = comp["total"] / (hbm * 1e9) * 1e3 / mean_ms
            if facts:
                roof["dram"]["overfetch_vs_compulsory"] = facts["dram_bytes_per_launch"] / comp["total"]
        except P.OOError as e:
            roof["compulsory"] = {"unavailable": str(e)}
        # camera -> RGB without the PCIe copy of the queries: primary visibility on the device + the query (12 B/query D2H only)
        if w.camera is not None:
            cam, sc = w.camera, w.scene
            ctx.oo_upload_scene(sc.spheres, sc.lo, sc.hi)
            qbuf = tuple(torch.empty((q.n, 3), dtype=torch.float32, device=dev) for _ in range(3))
            exd = ex

            def cam_to_rgb():
                ctx.oo_raycast(cam.eye, cam.look, cam.up, cam.vfov_deg, cam.width, cam.height, out=qbuf)
                ctx.oo_query(qbuf[0], qbuf[1], qbuf[2], exd, rgb=rgb)
                hrgb.copy_(rgb, non_blocking=True)
            for _ in range(3):
                cam_to_rgb()
            torch.cuda.synchronize(dev)
            tt = []
            for _ in range(e2e_steps):
                tc = time.perf_counter()
                cam_to_rgb()
                torch.cuda.synchronize(dev)
                tt.append((time.perf_counter() - tc) * 1e3)
            out["e2e_camera_to_rgb"] = {"ms_per_step": sum(tt) / len(tt), "value": q.n / (sum(tt) / len(tt) * 1e-3) / 1e6, "unit": UNIT,
                                        "h2d_bytes_per_step": 0, "d2h_bytes_per_step": int(12 * q.n),
                                        "api": "oo_raycast + oo_query + one D2H copy of the RGB: the frame's queries are made on the device (not the headline e2e: its inputs never cross PCIe)"}
    if world == 1 and not args.no_cpu_baseline and not args.quick:
        sample_q, sample_desc = oracle_sample(w, args.ref_sample)
        dt, threads = time_oracle(w, sample_q, repeats=3)
        sample_desc += "; best of 3"
        out["cpu_baseline"] = {"value": sample_q.n / dt / 1e6, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample_desc}
    # `frac` stays what the bench contract defines (algorithmic bytes / measured HBM peak) and can exceed 1 on a coherent frame, where
    # it is not a bound.  Beside it: the same number under an explicit name, and the tightest bound that does hold for this launch --
    # the largest of the times the compulsory bytes, the measured DRAM bytes, the issue slots and the MLP FLOPs need -- over the measured time.
    cand = {"mlp_flops": flop_time * 1e3}
    if isinstance(roof.get("compulsory"), dict) and "byte_time_ms" in roof["compulsory"]:
        cand["compulsory_bytes"] = roof["compulsory"]["byte_time_ms"]
    if "dram" in roof:
        cand["measured_dram_bytes"] = roof["dram"]["bytes_per_launch"] / (hbm * 1e9) * 1e3
    if "issue" in roof:
        cand["issue_slots"] = roof["issue"]["bound_ms"]
    tight = max(cand, key=cand.get)
    roof["frac_algorithmic"] = roof["frac"]
    roof["frac_tightest_bound"] = {"bound": tight, "bound_ms": cand[tight], "frac": cand[tight] / mean_ms, "candidates_ms": cand,
                                   "note": "a real lower bound on this launch's time over the measured time (<= 1 by construction); read this, "
                                           "not `frac`, when `frac` is above 1"}
    print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def run_sweep(args):
    """BASELINE.json configs[2] / configs[4] side measurements (not the headline line): one JSON line with a table.

    --sweep 2: config 2's frame in scanline order, Morton-sorted (oo_sort_queries; sort cost separate and included) and
               seeded-shuffled order.  --sweep 4: config 3's tree and MLP, batch sizes 2^16..2^24, coherent (screen-order
               hits of a 4096x4096 frame) and incoherent (area-weighted surface points, random order): encode-only and
               fused Mqueries/s against the roofline.  CUDA events on the launching stream, L2 flushed between launches."""
    import numpy as np
    import torch
    import gen
    import paper_2606_08469_b200 as P
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    hbm, tf, which = peaks()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)
    cu = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)

    def timed(fn, reps):
        for _ in range(3):
            flush.zero_()
            fn()
        evs = []
        for _ in range(reps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            evs.append((e0, e1))
        torch.cuda.synchronize(dev)
        t = sorted(a.elapsed_time(b) for a, b in evs)
        return t[len(t) // 2]

    rows = []
    if args.sweep == 2:
        w, desc = workload_for(2)
        q = w.queries
        ctx = P.OctaOctree(0).upload_workload(w)
        ctx.oo_reserve(q.n)
        ctx.oo_set_presort("none")                      # this table is about explicit orders
        x, nrm, wo, ex = cu(q.x), cu(q.nrm), cu(q.wo), cu(q.extra)
        rgb = torch.empty((q.n, 3), dtype=torch.float32, device=dev)
        perm = torch.empty(q.n, dtype=torch.int32, device=dev)
        shuf = cu(gen.shuffle_perm(q.n, 0).astype(np.int32))
        bq = desc["bytes_per_query"]
        t_scan = timed(lambda: ctx.oo_query(x, nrm, wo, ex, rgb=rgb), args.steps)
        t_sort = timed(lambda: ctx.oo_sort_queries(x, perm_out=perm), args.steps)
        t_sorted = timed(lambda: ctx.oo_query(x, nrm, wo, ex, perm=perm, rgb=rgb), args.steps)
        t_both = timed(lambda: (ctx.oo_sort_queries(x, perm_out=perm), ctx.oo_query(x, nrm, wo, ex, perm=perm, rgb=rgb)), args.steps)
        t_shuf = timed(lambda: ctx.oo_query(x, nrm, wo, ex, perm=shuf, rgb=rgb), args.steps)
        for name, t in (("scanline order", t_scan), ("morton-sorted (query only)", t_sorted), ("morton sort alone", t_sort),
                        ("sort + query, output in caller order", t_both), ("seeded random shuffle", t_shuf)):
            rows.append({"order": name, "ms": t, "Mqueries_per_s": q.n / t / 1e3, "roofline_frac": bq * q.n / (t * 1e-3) / 1e9 / hbm})
        out = {"sweep": "BASELINE.json configs[2]: query order on the 1280x720 frame", "workload": desc["workload"], "rows": rows}
    else:
        w = gen.scene_workload(3, seed=0, width=64, height=64)          # config 3's scene, tree, atlas and MLP
        L, F = len(w.tree.level_depth), w.atlas.F
        bq_fused = L * 4 * F * 2 + 48
        bq_enc = L * 4 * F * 2 + 24 + L * F * 2                           # x, wo in; features out
        ctx = P.OctaOctree(0).upload_workload(w)
        ctx.oo_set_presort("none")                      # the plain columns are the unsorted call; bin and auto have their own
        n_max = 1 << args.sweep_max_log2
        side = 1 << ((args.sweep_max_log2 + 1) // 2)
        cam = gen.make_camera(side, n_max // side, 0)
        dists = {}
        if args.sweep_dist in ("both", "coherent"):
            dists["coherent"] = gen.raycast(w.scene, cam)
        if args.sweep_dist in ("both", "incoherent"):
            dists["incoherent"] = gen.incoherent_queries(w.scene, n_max, 0)
        ctx.oo_reserve(n_max)
        feat = torch.empty((n_max, L * F), dtype=torch.float16, device=dev)
        rgb = torch.empty((n_max, 3), dtype=torch.float32, device=dev)
        perm = torch.empty(n_max, dtype=torch.int32, device=dev)
        floor = {}
        for dname, q in dists.items():
            X, Nn, W = cu(q.x), cu(q.nrm), cu(q.wo)
            # the latency floor of a call: ONE 128-query tile (launch + prologue + one descent/gather chain + the decoder's MMA
            # round trips, cold L2); no batch, however small, finishes sooner, so small batches are judged against it
            floor[dname] = {"fused_one_tile_ms": timed(lambda: ctx.oo_query(X[:128], Nn[:128], W[:128], rgb=rgb[:128]), 20),
                            "encode_one_tile_ms": timed(lambda: ctx.oo_encode(X[:128], W[:128], features=feat[:128]), 20)}
            for lg in range(args.sweep_min_log2, args.sweep_max_log2 + 1):
                n = 1 << lg
                x, nrm, wo = X[:n], Nn[:n], W[:n]
                reps = max(5, min(args.steps, (1 << 26) // n))
                t_f = timed(lambda: ctx.oo_query(x, nrm, wo, rgb=rgb[:n]), reps)
                t_e = timed(lambda: ctx.oo_encode(x, wo, features=feat[:n]), reps)
                row = {"distribution": dname, "n": n, "fused_ms": t_f, "fused_Mqueries_per_s": n / t_f / 1e3,
                       "fused_roofline_frac": bq_fused * n / (t_f * 1e-3) / 1e9 / hbm,
                       "encode_ms": t_e, "encode_Mqueries_per_s": n / t_e / 1e3,
                       "encode_roofline_frac": bq_enc * n / (t_e * 1e-3) / 1e9 / hbm}
                if dname == "incoherent":
                    # a1: Morton pre-sort inside the timed region, RGB still in the caller's order
                    t_s = timed(lambda: (ctx.oo_sort_queries(x, perm_out=perm[:n]),
                                         ctx.oo_query(x, nrm, wo, perm=perm[:n], rgb=rgb[:n])), reps)
                    row.update({"sort_plus_fused_ms": t_s, "sort_plus_fused_roofline_frac": bq_fused * n / (t_s * 1e-3) / 1e9 / hbm})
                # a1': OO_PRESORT_BIN, one counting pass inside oo_query / oo_encode that moves the queries (all launches timed;
                # min_queries=1 so that the table shows from which batch size on it pays)
                ctx.oo_set_presort("bin", min_queries=1)
                t_b = timed(lambda: ctx.oo_query(x, nrm, wo, rgb=rgb[:n]), reps)
                t_be = timed(lambda: ctx.oo_encode(x, wo, features=feat[:n]), reps)
                # the library's default: OO_PRESORT_AUTO at its default threshold (the warm-ups let it see the batch first)
                ctx.oo_set_presort("auto")
                t_a = timed(lambda: ctx.oo_query(x, nrm, wo, rgb=rgb[:n]), reps)
                auto_binned = bool(ctx.oo_get_info()["presorted_last_query"])
                t_ae = timed(lambda: ctx.oo_encode(x, wo, features=feat[:n]), reps)
                ctx.oo_set_presort("none")
                row.update({"bin_fused_ms": t_b, "bin_fused_roofline_frac": bq_fused * n / (t_b * 1e-3) / 1e9 / hbm,
                            "bin_encode_ms": t_be, "bin_encode_roofline_frac": bq_enc * n / (t_be * 1e-3) / 1e9 / hbm,
                            "auto_fused_ms": t_a, "auto_fused_roofline_frac": bq_fused * n / (t_a * 1e-3) / 1e9 / hbm, "auto_binned": auto_binned,
                            "auto_encode_ms": t_ae, "auto_encode_roofline_frac": bq_enc * n / (t_ae * 1e-3) / 1e9 / hbm})
                rows.append(row)
        out = {"sweep": "BASELINE.json configs[4]: batch size x query distribution on the config-3 tree and MLP",
               "tree_nodes": w.tree.n_nodes, "atlas_bytes": w.atlas.nbytes, "bytes_per_query": {"fused": bq_fused, "encode": bq_enc},
               "latency_floor": floor, "rows": rows}
    out.update({"unit": UNIT, "l2": "flushed between launches (256 MB memset)", "timing": "median of CUDA-event times",
                "peak_gbs": hbm, "peak_source": which, "data": "synthetic"})
    print(json.dumps(out))
    return 0


def run_raycast(args):
    """--sweep 5: primary visibility on the device: oo_raycast alone, and camera -> RGB
    (oo_raycast + oo_query, no host copy of the queries), for config 1's and config 3's frames."""
    import numpy as np
    import torch
    import gen
    import paper_2606_08469_b200 as P
    from oracle import oo_raycast as RC
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def timed(fn, reps):
        for _ in range(3):
            flush.zero_()
            fn()
        evs = []
        for _ in range(reps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            evs.append((e0, e1))
        torch.cuda.synchronize(dev)
        t = sorted(a.elapsed_time(b) for a, b in evs)
        return t[len(t) // 2]

    rows = []
    for cfg in (1, 3):
        w, desc = workload_for(cfg)
        cam, sc = w.camera, w.scene
        ctx = P.OctaOctree(0).upload_workload(w)
        ctx.oo_set_presort("none")
        ctx.oo_upload_scene(sc.spheres, sc.lo, sc.hi)
        n = cam.width * cam.height
        out = tuple(torch.empty((n, 3), dtype=torch.float32, device=dev) for _ in range(3))
        rgb = torch.empty((n, 3), dtype=torch.float32, device=dev)
        cast = lambda: ctx.oo_raycast(cam.eye, cam.look, cam.up, cam.vfov_deg, cam.width, cam.height, out=out)
        t_c = timed(cast, args.steps)
        t_q = timed(lambda: ctx.oo_query(out[0], out[1], out[2], rgb=rgb), args.steps)
        t_b = timed(lambda: (cast(), ctx.oo_query(out[0], out[1], out[2], rgb=rgb)), args.steps)
        n_surf = len(sc.spheres) + 5
        row = {"config": cfg, "frame": "%dx%d" % (cam.width, cam.height), "surfaces": n_surf, "raycast_ms": t_c, "query_ms": t_q,
               "raycast_plus_query_ms": t_b, "Mrays_per_s": n / t_c / 1e3, "camera_to_rgb_Mqueries_per_s": n / t_b / 1e3,
               "ray_surface_tests_per_s": n * n_surf / (t_c * 1e-3), "bytes_written_per_ray": 36}
        if not args.no_cpu_baseline and not args.quick:
            rws = np.arange(0, cam.height, 32)
            t0 = time.perf_counter()
            RC.raycast(sc.spheres, sc.lo, sc.hi, cam.eye, cam.look, cam.up, cam.vfov_deg, cam.width, cam.height, rows=rws)
            dt = time.perf_counter() - t0
            row["cpu_oracle_Mrays_per_s"] = len(rws) * cam.width / dt / 1e6
        rows.append(row)
        ctx.close()
    print(json.dumps({"sweep": "primary visibility on the device (f5): oo_raycast, fp64 arithmetic, one thread per pixel", "rows": rows,
                      "l2": "flushed between launches (256 MB memset)", "timing": "median of CUDA-event times", "data": "synthetic",
                      "cpu_oracle": "oracle/oo_raycast.py (numpy float64, 1 core) on every 32nd scanline"}))
    return 0


def run_full(args):
    """--sweep 8: the paper's FULL query at the paper's own shapes: 8 consecutive levels
    (depths 2..9), C = 4 fp32 vertex maps of resolution 2^8+1 .. 2^1+1, 8-neighbour trilinear blend, disparity-shifted
    mirror direction, Eq. 12 attributes, decoder 4 x 128, one 1024x1024 frame of primary hits; then each piece switched
    off in turn.  One JSON line with a table (not the headline line)."""
    import numpy as np
    import torch
    import gen
    import paper_2606_08469_b200 as P
    from oracle import oo_oracle_full as FO
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    hbm, tf, which = peaks()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)
    cu = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    w = gen.paper_workload(seed=0)
    q, disp = w.queries, w.meta["disparity"]
    L, F = len(w.tree.level_depth), w.atlas.F
    ctx = P.OctaOctree(0)
    ctx.oo_set_presort("none")
    ctx.oo_upload_tree(w.tree, w.atlas.levels, w.atlas.dtype, dirmap="vertex")
    x, nrm, wo, ex, dd = cu(q.x), cu(q.nrm), cu(q.wo), cu(q.extra), cu(disp)
    rgb = torch.empty((q.n, 3), dtype=torch.float32, device=dev)
    feat_rows = []

    def timed(fn, reps, do_flush=True):
        for _ in range(3):
            flush.zero_()
            fn()
        evs = []
        for _ in range(reps):
            if do_flush:
                flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            evs.append((e0, e1))
        torch.cuda.synchronize(dev)
        t = sorted(a.elapsed_time(b) for a, b in evs)
        return t[len(t) // 2]

    variants = [("full: trilinear8 + vertex + shifted + Eq.12 attrs, 4x128", "trilinear8", "shifted", "paper", 128),
                ("no shift (mirror direction for every cell)", "trilinear8", "mirror", "paper", 128),
                ("nearest cell (P:266 ablation)", "nearest", "shifted", "paper", 128),
                ("nearest cell, mirror direction", "nearest", "mirror", "paper", 128),
                ("full gather, decoder 4x64", "trilinear8", "shifted", "paper", 64)]
    rows = []
    if args.quick:
        variants = variants[:1]
    for name, spatial, lookup, attrs, width in variants:
        mlp = gen.make_mlp(L * F + 13, 4, 0, width=width)
        ctx.oo_upload_mlp(mlp.weights, mlp.out_act)
        ctx.oo_set_mode(spatial, lookup, attrs)
        # live neighbours (non-empty cells inside the grid) decide the bytes the method must read
        sub = slice(0, q.n, 16)
        _, s, _ = ctx.oo_encode_full(x[sub].contiguous(), nrm[sub].contiguous(), wo[sub].contiguous(), dd[sub].contiguous(), want_debug=True)
        live = float((s >= 0).float().sum(dim=(1, 2)).mean())
        J = 8 if spatial == "trilinear8" else 1
        bq = live * 3 * F * 4 + 36 + 4 + 16 + 12
        dims = [L * F + 13] + [width] * 4 + [3]
        flops = 2 * sum(a * b for a, b in zip(dims[:-1], dims[1:]))
        t = timed(lambda: ctx.oo_query(x, nrm, wo, ex, rgb=rgb, disparity=dd), args.steps)
        tw = t if args.quick else timed(lambda: ctx.oo_query(x, nrm, wo, ex, rgb=rgb, disparity=dd), min(args.steps, 20), do_flush=False)
        te = None if args.quick else timed(lambda: ctx.oo_encode_full(x, nrm, wo, dd), min(args.steps, 20))
        rows.append({"variant": name, "ms": t, "ms_warm_l2": tw, "Mqueries_per_s": q.n / t / 1e3, "encode_only_ms": te,
                     "live_neighbour_lookups_per_query": live, "of": L * J, "algorithmic_bytes_per_query": bq,
                     "flop_per_query": flops, "byte_time_ms": bq * q.n / (hbm * 1e9) * 1e3, "flop_time_ms": flops * q.n / (tf * 1e12) * 1e3,
                     "roofline_frac": max(bq * q.n / (hbm * 1e9), flops * q.n / (tf * 1e12)) / (t * 1e-3)})
    # Eq. 7 on the device: the disparity predictor alone, then the full query predicting d^ itself (two launches, no d^ input)
    net = gen.make_disparity_net(0)
    ctx.oo_upload_disparity(net.res, net.hash_log2, net.tables, net.weights)
    ctx.oo_reserve(q.n)
    mlp = gen.make_mlp(L * F + 13, 4, 0, width=128)
    ctx.oo_upload_mlp(mlp.weights, mlp.out_act)
    ctx.oo_set_mode("trilinear8", "shifted", "paper")
    dbuf = torch.empty(q.n, dtype=torch.float32, device=dev)
    G = len(net.res)
    t_p = timed(lambda: ctx.oo_predict_disparity(x, nrm, wo, disparity=dbuf), args.steps)
    t_pq = timed(lambda: ctx.oo_query(x, nrm, wo, ex, rgb=rgb), args.steps)
    bq_p = G * 8 * 4 + 36 + 4
    fl_p = 2 * ((2 * G + 3) * 64 + 64 * 64 + 64)
    disparity_rows = [
        {"variant": "disparity predictor g_psi alone (Eq. 7): %d-level hash grid %s, 2^%d-entry tables (%.1f MB), MLP %d->2x64->1 exp" %
                    (G, net.res, net.hash_log2, sum(t.nbytes for t in net.tables) / 1e6, 2 * G + 3),
         "ms": t_p, "Mqueries_per_s": q.n / t_p / 1e3, "algorithmic_bytes_per_query": bq_p, "flop_per_query": fl_p,
         "byte_time_ms": bq_p * q.n / (hbm * 1e9) * 1e3, "roofline_frac": bq_p * q.n / (hbm * 1e9) / (t_p * 1e-3)},
        {"variant": "full query predicting d^ itself (g_psi launch + fused full-query launch)", "ms": t_pq, "Mqueries_per_s": q.n / t_pq / 1e3}]
    rows += disparity_rows
    out = {"sweep": "full query at the paper's shapes (PAPER.md implementation details; SURVEY.md 8(f) f1-f4)",
           "workload": "1024x1024 primary hits of the three-sphere scene; octree depth 9 (%d nodes), used depths %s, vertex maps R_l+1 = %s, C=%d fp32 (%.0f MB), "
                       "Eq. 12 attributes (13 scalars), synthetic disparity U(0.25,4)" %
                       (w.tree.n_nodes, w.tree.level_depth, [r + 1 for r in w.tree.level_res], F, w.atlas.nbytes / 1e6),
           "rows": rows, "unit": UNIT, "l2": "flushed between launches (256 MB memset)", "timing": "median of CUDA-event times",
           "peak_gbs": hbm, "peak_tflops": tf, "peak_source": which, "data": "synthetic",
           "paper_context": "Table 1: 10-20 ms per frame on an RTX 3090 including Mitsuba G-buffer extraction and the disparity network (not comparable)"}
    if not args.no_cpu_baseline and not args.quick:
        n_s = 16384
        idx = np.arange(0, q.n, q.n // n_s)[:n_s]
        qs = q.take(idx)
        mode = FO.Mode("trilinear8", "vertex", "shifted", "paper")
        mlp = gen.make_mlp(L * F + 13, 4, 0, width=128)
        t0 = time.perf_counter()
        FO.query_full(w.tree, w.atlas.levels, mlp.weights, qs.x, qs.nrm, qs.wo, qs.extra, "exp", mode, disp[idx])
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": n_s / dt / 1e6, "unit": UNIT, "cores": 1, "kind": "oracle (numpy float64, oo_oracle_full.py)",
                               "sample": "%d queries (every %dth pixel)" % (n_s, q.n // n_s)}
    print(json.dumps(out))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[1, 2, 3, 4], help="BASELINE.json configs[k]; 4 = its incoherent distribution at 2^22 queries")
    ap.add_argument("--path", default="auto", choices=["auto", "mma", "tc", "tm", "unfused", "generic"])
    ap.add_argument("--ref-sample", type=int, default=1 << 22, help="queries in the cpu_baseline sample (capped at the frame)")
    ap.add_argument("--ref-budget", type=float, default=90.0, help="--impl reference: seconds of CPU work the W + K steps may take")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", type=int, default=0, choices=[0, 2, 4, 5, 8], help="side measurements of configs[2] / configs[4] / (8) the paper's full query at its own shapes (a table, not the headline line)")
    ap.add_argument("--sweep-max-log2", type=int, default=24)
    ap.add_argument("--sweep-min-log2", type=int, default=16)
    ap.add_argument("--sweep-dist", default="both", choices=["both", "coherent", "incoherent"])
    ap.add_argument("--presort", default="auto", choices=["auto", "none", "bin"], help="oo_set_presort for the run (default: the library's own default, auto)")
    ap.add_argument("--quick", action="store_true", help="timed region only (no warm-L2 / e2e / CPU legs): the command ncu wraps")
    ap.add_argument("--phase", default="fused", choices=["fused", "encode"], help="fused = the whole hot path (the headline); encode = oo_encode alone (a2-a6), a side measurement and the ncu target for the encoding phase")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"], help="N > 1: every rank its own frame (weak) or one frame split across ranks + RGB all-gather (strong)")
    ap.add_argument("--dry-run-dist", action="store_true", help="the N > 1 host logic on CPU with gloo (launcher, sharding, gather, reductions): what the CPU tests drive; measures nothing")
    ap.add_argument("--ingest-ncu", default=None, help="ncu --csv launch list to store in profiles/traffic.json for --config (see ingest_ncu)")
    ap.add_argument("--ingest-kernel", default="fused", help="substring of the dominant kernel's name for --ingest-ncu")
    args = ap.parse_args()
    if args.ingest_ncu:
        return ingest_ncu(args)
    if args.impl == "ours" and not args.sweep:
        rc = relaunch_if_needed(args)
        if rc >= 0:
            return rc
        if args.dry_run_dist:
            return run_dry_dist(args)
    if args.sweep == 8:
        return run_full(args)
    if args.sweep == 5:
        return run_raycast(args)
    if args.sweep:
        return run_sweep(args)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
