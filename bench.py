#!/usr/bin/env python
"""bench.py — BASELINE.json's metric on BASELINE.json's workload.

Metric: track-steps/s (and step-kernel HBM GB/s as a fraction of the measured B200 peak) on the
single-step microbenchmark (BASELINE.json configs[2]): 2^24 tracks, 40 % e- / 10 % e+ / 50 % gamma,
uniform in the 50-layer Pb/lAr calorimeter, isotropic, log-uniform 100 keV - 10 GeV, exp(1)
interaction lengths; one adept_step per "step", dense double buffer, per layout.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--layout soa|aos|aosoa32|aosoa64|soa16|all] [--impl reference]

`--gpus N` with N > 1 and no torchrun environment re-launches itself as N ranks (torch.distributed.run,
rendezvous on 127.0.0.1); under torchrun it uses the ranks it was given.  `n_gpus` is the number of
ranks that actually ran.

The default line also carries, beside the headline (rank 0, one GPU): `showers` = BASELINE.json
configs[1] ("full") and configs[4] ("heavy") through adept_inject + adept_run, each with the oracle
timed on the same workload and the full-size parity of its counts and per-layer deposits; and
`sweep` = configs[3], per scheme x layout x occupancy the step time, its roofline fraction and the
time of slot allocation / compaction (section clocks of the timing variant of the library).
`--extras none` prints the headline only.

One JSON line on stdout (rank 0).  `value` is measured with the tracks resident in HBM: every timed
step starts from a pristine copy of the workspace (restored outside the timed region, L2 flushed) and
is timed with CUDA events on the stream the kernel is launched on.  `e2e` is the same step through
the C ABI with HOST buffers: adept_load_tracks (H2D) + adept_step + adept_read_tracks (D2H) inside
the timed region.  `cpu_baseline` / `--impl reference` time the oracle (oracle/, single thread) on
the host cores; that is the only use of oracle/ here.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import CONFIGS, gen_tracks, geometry_for, tables_for  # noqa: E402

WORKLOAD = "single_step"
RECORD_BYTES = {"aos": 64, "soa": 56, "aosoa32": 56, "aosoa64": 56, "soa16": 56, "aosoa16": 56, "aosoa128": 56, "hc16": 56, "aosoa8": 56}     # bytes per record per layout
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_traffic.csv")


EXTRAS_FILE = os.path.join(ROOT, "bench_extras.json")
LINE_LIMIT = 8192          # bytes: the driver keeps a bounded tail of stdout and parses its last JSON line


def _r(x, digits=5):
    """Floats of the compact line to `digits` significant digits (the full values are in the extras file)."""
    if isinstance(x, float):
        return float("%.*g" % (digits, x))
    if isinstance(x, (list, tuple)):
        return [_r(v, digits) for v in x]
    if isinstance(x, dict):
        return {k: _r(v, digits) for k, v in x.items()}
    return x


def contract_line(out: dict) -> dict:
    """The one JSON line the driver parses, from the full result `out`: the contract keys unchanged, and of
    the bulky extras (per-layout detail, shower blocks with their 50-bin deposits, the sweep's 40 cells with
    per-field counts) only scalar summaries and short arrays.  Everything else goes to EXTRAS_FILE."""
    keep = ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
            "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "e2e", "roofline", "cpu_baseline",
            "parity_full_size")
    line = {k: out[k] for k in keep if k in out}
    if "layouts" in out:
        line["layouts_ms_per_step"] = {l: _r(v["ms_per_step"]) for l, v in out["layouts"].items()}
    if "single_step_physics" in out:
        line["single_step_physics"] = _r(out["single_step_physics"])
    if "showers" in out:
        sh = {}
        for name, b in out["showers"].items():
            e = {k: b[k] for k in ("value", "ms_per_run", "ms_min", "iterations", "track_steps", "us_per_iteration",
                                   "showers_per_s", "layout", "scheme", "same_counts_as_dense", "scaling") if k in b}
            if "parity_full_size" in b:
                e["counts_bit_exact"] = b["parity_full_size"]["counts_bit_exact"]
                e["edep_layer_rel_err"] = b["parity_full_size"]["edep_layer_rel_err"]
            if "cpu_baseline" in b:
                e["cpu_value"] = b["cpu_baseline"]["value"]
            sh[name] = _r(e)
        line["showers"] = sh
    if "sweep" in out:
        sw = out["sweep"]
        cells = sw["cells"]
        occs = sorted({c["occupancy"] for c in cells})
        lays = []
        for c in cells:
            if c["layout"] not in lays:
                lays.append(c["layout"])
        summ = {"workload": "BASELINE.json configs[3]", "best": _r(sw["best"]), "occupancies": occs, "layouts": lays}
        for scheme in ("dense", "sparse"):
            sc = [c for c in cells if c["scheme"] == scheme]
            if not sc:
                continue
            at = {(c["layout"], c["occupancy"]): c for c in sc}
            grid = lambda f: [[_r(f(at[(l, o)]), 4) if (l, o) in at else None for o in occs] for l in lays]
            blk = {"ms_per_step": grid(lambda c: c["ms_per_step"]),
                   "roofline_frac": grid(lambda c: c["roofline"]["frac"])}
            if any("alloc_compaction_ms" in c for c in sc):
                blk["alloc_compaction_ms"] = grid(lambda c: c.get("alloc_compaction_ms"))
            counted = [c for c in sc if "field_reads" in c]
            if counted:
                # BASELINE.json configs[3] "per-field read/write counts" (Fig. 5): one instrumented
                # cell per layout of this scheme, fields in the order of `field_names`
                # cell per scheme in the line (the other layouts' counts are in the extras file), fields in the order
                # of `field_names`; and per counted layout the 128-byte lines touched over the method's own bytes
                c0 = ([c for c in counted if c["layout"] == "aosoa32"] or counted)[0]
                blk["field_counts"] = {"layout": c0["layout"], "occupancy": c0["occupancy"],
                                       "reads": list(c0["field_reads"].values()), "writes": list(c0["field_writes"].values())}
                blk["line_bytes_over_algorithmic"] = {c["layout"]: _r(c.get("line_bytes_over_algorithmic"), 4) for c in counted}
                summ["field_names"] = list(c0["field_reads"].keys())
            summ[scheme] = blk
        line["sweep"] = summ
    if "extras_file" in out:
        line["extras_file"] = out["extras_file"]
    return line


def emit(out: dict) -> None:
    """Write the full result to EXTRAS_FILE and print the compact contract line as the LAST line of stdout."""
    try:
        with open(EXTRAS_FILE, "w") as f:
            json.dump(out, f)
        out["extras_file"] = os.path.basename(EXTRAS_FILE)
    except OSError as e:   # a read-only checkout: the line still goes out
        sys.stderr.write("bench.py: could not write %s (%s)\n" % (EXTRAS_FILE, e))
    text = json.dumps(contract_line(out), separators=(",", ":"))
    if len(text) > LINE_LIMIT:   # never let an extra push the contract keys out of the driver's view
        slim = contract_line({k: v for k, v in out.items() if k not in ("sweep", "showers", "layouts")})
        slim["note"] = "extras dropped from the line (over %d bytes); see extras_file" % LINE_LIMIT
        text = json.dumps(slim, separators=(",", ":"))
    sys.stderr.flush()
    sys.stdout.write(text + "\n")
    sys.stdout.flush()


def ncu_traffic(workload: str, layout: str, scheme: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one step_kernel launch, from the committed table
    of `ncu --set full` captures (profiles/ncu_traffic.csv; the .md beside it names the commands).
    Returns (bytes, source) or (None, None) when no capture exists for this kernel and workload."""
    try:
        with open(TRAFFIC_CSV) as f:
            rows = [l.strip().split(",") for l in f if l.strip() and not l.startswith("#")]
    except OSError:
        return None, None
    head, best = rows[0], None
    for r in rows[1:]:
        d = dict(zip(head, r))
        if d["workload"] == workload and d["layout"] == layout and d["scheme"] == scheme:
            best = d                                   # later rows are later captures
    if best is None:
        return None, None
    # the capture is of the kernels as they were then: say so when csrc/ has changed since (rows older than
    # round 3 carry no source hash and count as stale)
    fresh = best.get("csrc_sha") and best["csrc_sha"] == csrc_sha()
    return float(best["dram_bytes_read"]) + float(best["dram_bytes_write"]), \
        "profiles/ncu_traffic.csv (%s, commit %s%s)" % (best["capture"], best["commit"],
                                                        "" if fresh else "; STALE: csrc/ changed since the capture")


def csrc_sha() -> str:
    """Hash of the kernel sources, as recorded beside each ncu capture in profiles/ncu_traffic.csv."""
    import glob
    import hashlib
    h = hashlib.sha1()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2302_08252_b200", "csrc", "*"))):
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def measured_peak():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (profiling recipe's clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        # under load = the upper half of the samples (idle gaps between steps pull the clock down)
        sm.sort()
        load = sm[len(sm) // 2:] if sm else []
        return {"sm_mhz": float(np.median(load)) if load else None,
                "sm_max_mhz": max(smax) if smax else None, "reasons": sorted(reasons), "samples": len(sm)}


def population(n_tracks: int, rank: int):
    c = CONFIGS[WORKLOAD]
    return gen_tracks(n_tracks, c["seed"] + 1000 * rank, geometry_for(WORKLOAD), c["e_max"], c["fractions"])


def oracle_single_step(pop, sample_tracks: int, want_tracks: bool = False, physics: int = 0):
    """Time the oracle, as it stands, on the first `sample_tracks` tracks of each kind's share."""
    from oracle import Oracle
    c = CONFIGS[WORKLOAD]
    total = sum(p.shape[0] for p in pop)
    frac = min(1.0, sample_tracks / total)
    o = Oracle(geometry_for(WORKLOAD), tables_for(WORKLOAD, physics), seed=c["seed"])
    n = 0
    for k in range(3):
        m = int(round(pop[k].shape[0] * frac))
        o.load_tracks(k, pop[k][:m])
        n += m
    t0 = time.perf_counter()
    o.step()
    dt = time.perf_counter() - t0
    r = o.result()
    if want_tracks:
        r["tracks"] = [by_id(o.read_tracks(k, pop[0].dtype)) for k in range(3)]
    o.close()
    return n, dt, r


def by_id(tracks):
    """All tracks in id order: the full-size parity check compares every one of them word for word."""
    key = tracks["id_hi"].astype(np.uint64) << np.uint64(32) | tracks["id_lo"].astype(np.uint64)
    return tracks[np.argsort(key, kind="stable")]


def full_size_parity(gpu: dict, ref: dict) -> dict:
    """Every output track of the GPU step against the oracle's (both in id order), word for word.
    Discrete-branch disagreements (north_star: to be reported): a track that took another branch on the GPU
    has another fate -- it is missing, extra, or of another kind in the output.  north_star allows them only
    where the oracle's decision margin is below 1e-6; with none at all, none has a larger margin."""
    keys = ("steps", "secondaries", "killed", "escaped_n", "live")
    n_cmp = n_missing = n_diff = 0
    for a, b in zip(gpu["tracks"], ref["tracks"]):
        ka = a["id_hi"].astype(np.uint64) << np.uint64(32) | a["id_lo"].astype(np.uint64)
        kb = b["id_hi"].astype(np.uint64) << np.uint64(32) | b["id_lo"].astype(np.uint64)
        common = np.intersect1d(ka, kb)
        n_missing += int(ka.shape[0] + kb.shape[0] - 2 * common.shape[0])
        aa, bb = a[np.isin(ka, common)], b[np.isin(kb, common)]
        n_cmp += int(common.shape[0])
        n_diff += int((aa.view(np.uint8).reshape(-1, 56) != bb.view(np.uint8).reshape(-1, 56)).any(axis=1).sum())
    return {"counts_bit_exact": bool(all((gpu[k] == ref[k]).all() for k in keys)),
            "tracks_compared": n_cmp, "tracks_with_another_fate": n_missing,
            "tracks_with_any_word_differing": n_diff,
            "branch_disagreement_rate": (n_missing / max(1, n_cmp)),
            "disagreements_with_margin_ge_1e-6": 0 if n_missing == 0 else None,   # None: would need the oracle's trace
            "edep_rel_err": float(np.max(np.abs(gpu["edep_layer"] - ref["edep_layer"]) / np.maximum(ref["edep_layer"], 1e-30)))}


def host_cores() -> int:
    return os.cpu_count() or 1


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle on the host cores, same metric/config, bounded sample per step.
    Under torchrun rank 0 alone runs and prints; the other ranks exit without work."""
    if rank != 0:
        return
    sample = min(args.tracks, 1 << 21)
    pop = population(sample, 0)
    for _ in range(args.warmup):
        oracle_single_step(pop, sample)
    n_tot, t_tot = 0, 0.0
    for _ in range(args.steps):
        n, dt, _ = oracle_single_step(pop, sample)
        n_tot += n
        t_tot += dt
    v = n_tot / t_tot
    cpu = {"value": v, "unit": "track-steps/s", "cores": 1, "host_cores": host_cores(), "kind": "oracle",
           "sample": "one adept_step-equivalent oracle iteration over %d tracks of the config-3 population per step" % sample}
    print(json.dumps({
        "impl": "reference", "metric": "track-steps/sec", "value": v, "unit": "track-steps/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "single-step microbenchmark (BASELINE.json configs[2]), oracle on host, "
                               "%d-track sample per step" % sample},
        "cpu_baseline": cpu,
        "e2e": {"value": v, "unit": "track-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def bench_layout(ctx, torch, pop, steps, warmup, flush, barrier):
    """Device-resident timing of adept_step: returns per-step ms list and the counts after one step."""
    for k in range(3):
        ctx.load_tracks(k, pop[k])
    torch.cuda.synchronize()
    pristine = ctx.snapshot()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]

    def one(e0, e1):
        ctx.rewind(pristine)                   # include/adept.h "Workspace", untimed
        flush.zero_()                          # L2 flush: 256 MiB > 126 MB L2, untimed
        if e0 is not None:
            e0.record(ctx.stream)
        ctx.step(sync=False)
        if e1 is not None:
            e1.record(ctx.stream)

    for _ in range(warmup):
        one(None, None)
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    for e0, e1 in ev:
        one(e0, e1)
    torch.cuda.synchronize()
    barrier()
    wall = time.perf_counter() - t0
    ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    res = ctx.result()
    res["tracks"] = [by_id(ctx.read_tracks(k)) for k in range(3)]
    del pristine
    return ms, res, wall


def run_gpu(args, rank: int, world: int, local_rank: int):
    import torch
    from paper_2302_08252_b200 import Context
    from paper_2302_08252_b200.binding import TRACK_DTYPE
    dist = None
    # Test hook (tests/test_bench_contract.py): ADEPT_BENCH_ONE_DEVICE=1 runs every rank on cuda:0 with
    # the gloo backend, to exercise the N > 1 plumbing on a one-GPU box.  The ranks' kernels never wait
    # on one another (the only exchanges are host-side barriers and all-reduces), so this is a test of
    # the code path, not a measurement.
    one_device = os.environ.get("ADEPT_BENCH_ONE_DEVICE") == "1"
    if one_device:
        local_rank = 0
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        if one_device:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    def barrier():
        if dist is not None:
            dist.barrier()

    def max_over_ranks(x: float) -> float:
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cpu" if one_device else dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    geo, tab = geometry_for(WORKLOAD), tables_for(WORKLOAD)
    n_tracks = args.tracks
    pop = population(n_tracks, rank)                       # weak scaling: each rank its own 2^24 tracks
    biggest = max(p.shape[0] for p in pop)
    capacity = int(biggest * 1.25) + 4096                  # one step grows the photon set by ~16 %
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    layouts = ["aosoa32", "aosoa64", "soa16", "hc16", "soa", "aos"] if args.layout == "all" else [args.layout]
    per_layout, results = {}, {}
    sampler = ClockSampler(local_rank)
    sampler.start()
    for layout in layouts:
        ctx = Context(geo, tab, layout=layout, scheme="dense", capacity=capacity,
                      seed=CONFIGS[WORKLOAD]["seed"], device="cuda:%d" % local_rank)
        ms, res, wall = bench_layout(ctx, torch, pop, args.steps, args.warmup, flush, barrier)
        total_ms = max_over_ranks(float(np.sum(ms)))
        n_out = int(res["live"].sum())
        bytes_per_launch = RECORD_BYTES[layout] * (n_tracks + n_out)
        per_layout[layout] = {
            "ms_per_step": total_ms / args.steps, "ms_min": float(np.min(ms)), "ms_median": float(np.median(ms)),
            "track_steps_per_s": world * n_tracks * args.steps / (total_ms * 1e-3),
            "algorithmic_bytes_per_launch": bytes_per_launch,
            "algorithmic_GBps": bytes_per_launch / (float(np.mean(ms)) * 1e-3) / 1e9,
            "survivors_plus_secondaries": n_out}
        results[layout] = res
        ctx.destroy()
        del ctx
        torch.cuda.empty_cache()
    clocks = sampler.stop()
    # headline = AoSoA-32, the layout whose ncu captures are under profiles/ (AoSoA-64 and SoA16 are
    # within 1 % of it, run to run); another layout takes over only if it is clearly faster
    main = layouts[0]
    best = min(per_layout, key=lambda l: per_layout[l]["ms_per_step"])
    if per_layout[best]["ms_per_step"] < 0.97 * per_layout[main]["ms_per_step"]:
        main = best
    main_res = results[main]

    # ---- e2e: host buffers, H2D + step + D2H inside the timed region (main layout) ----------
    ctx = Context(geo, tab, layout=main, scheme="dense", capacity=capacity,
                  seed=CONFIGS[WORKLOAD]["seed"], device="cuda:%d" % local_rank)
    pinned_in = [torch.from_numpy(p.view(np.uint8).copy()).pin_memory() for p in pop]
    host_in = [t.numpy().view(TRACK_DTYPE) for t in pinned_in]
    pinned_out = [torch.empty(capacity * 56, dtype=torch.uint8).pin_memory() for _ in range(3)]
    host_out = [t.numpy().view(TRACK_DTYPE) for t in pinned_out]
    e2e_steps = max(1, min(args.steps, 10))
    e2e_t, d2h, e2e_each = 0.0, 0, []
    for it in range(1 + e2e_steps):                        # first pass is a warm-up
        ctx.reset()
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for k in range(3):
            ctx.load_tracks(k, host_in[k])
        counts = ctx.step()
        d2h = 0
        for k in range(3):
            d2h += 56 * ctx.read_tracks(k, out=host_out[k])
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0)
        if it > 0:
            e2e_t += dt
            e2e_each.append(dt)
    # the same with only the step's counts read back (tracks stay on the device for the next
    # iteration, as they do inside adept_run): reported beside the full round trip
    e2e_c = 0.0
    for it in range(1 + e2e_steps):
        ctx.reset()
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for k in range(3):
            ctx.load_tracks(k, host_in[k])
        counts = ctx.step()
        dt = max_over_ranks(time.perf_counter() - t0)
        if it > 0:
            e2e_c += dt
    ctx.destroy()
    del ctx, pinned_in, pinned_out, host_in, host_out
    e2e_value = world * n_tracks * e2e_steps / e2e_t
    e2e_counts_only = world * n_tracks * e2e_steps / e2e_c

    # ---- N > 1: the event-sharded heavy showers beside the weak-scaled step ----
    sharded = None
    if world > 1 and "showers" in args.extras:
        sharded = sharded_showers(args, "heavy" if "heavy" in args.extras else "full", rank, world, local_rank, dist,
                                  max_over_ranks, reduce_on_cpu=one_device)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peak()
    m = per_layout[main]
    full_size = n_tracks == CONFIGS[WORKLOAD]["n_tracks"]
    traffic, traffic_src = ncu_traffic("single_step", main, "dense") if full_size else (None, None)
    shape = "1024 threads x 1 CTA/SM" if n_tracks >= (1 << 22) else "256 threads x 4 CTAs/SM"   # adept_api.cu launch_iteration
    out = {
        "metric": "track-steps/sec", "value": m["track_steps_per_s"], "unit": "track-steps/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": m["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "single-step microbenchmark (BASELINE.json configs[2]): %d tracks per GPU, "
                               "40/10/50 %% e-/e+/gamma, one adept_step, dense double buffer" % n_tracks,
                   "layout": main, "scheme": "dense", "tracks_per_gpu": n_tracks, "capacity_per_kind": capacity,
                   "parallelism": "independent track shards, no collective" if world > 1 else "single GPU",
                   "l2": "workspace restored from a pristine copy and 256 MiB written between timed steps; "
                         "inputs (0.94 GB) exceed L2"},
        "clocks": clocks,
        "gpu_launches": args.steps,
        "e2e": {"value": e2e_value, "unit": "track-steps/s", "h2d_bytes_per_step": 56 * n_tracks,
                "d2h_bytes_per_step": d2h + 512, "steps": e2e_steps,
                "ms_min": 1e3 * float(np.min(e2e_each)), "ms_median": 1e3 * float(np.median(e2e_each)),
                "counts_only": {"value": e2e_counts_only, "unit": "track-steps/s", "d2h_bytes_per_step": 512,
                                "what": "adept_load_tracks x3 + adept_step with its adept_counts read back"},
                "what": "adept_load_tracks x3 (pinned host) + adept_step + adept_read_tracks x3"},
        "roofline": {"bound": "hbm", "achieved": m["algorithmic_GBps"], "peak": peak, "unit": "GB/s",
                     "frac": m["algorithmic_GBps"] / peak,
                     "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": peak_src,
                     "kernel": "adept::step_kernel<%s, dense, %s>" % (main, shape),
                     "bytes_per_launch": m["algorithmic_bytes_per_launch"]},
        "layouts": per_layout,
    }
    if sharded is not None:
        out["showers"] = {("heavy" if "heavy" in args.extras else "full") + "_sharded": sharded}
    if world == 1 and not args.no_cpu:
        n, dt, r = oracle_single_step(pop, n_tracks, want_tracks=True)
        out["cpu_baseline"] = {"value": n / dt, "unit": "track-steps/s", "cores": 1, "host_cores": host_cores(),
                               "kind": "oracle",
                               "sample": "one oracle iteration over all %d tracks of the same population" % n,
                               "seconds": dt}
        out["parity_full_size"] = full_size_parity(main_res, r)
        del r
    del main_res, results
    torch.cuda.empty_cache()
    if world == 1 and "physics" in args.extras:
        # the same step under the extended rule sets (DESIGN.md rules X36-X39): physics 2
        # reads and writes the paper's three cold fields of every e+- in a side array, 12 B
        out["single_step_physics"] = {}
        n_epm = pop[0].shape[0] + pop[1].shape[0]
        for physics in (1, 2):
            ctx = Context(geo, tables_for(WORKLOAD, physics), layout=main, scheme="dense", capacity=capacity,
                          seed=CONFIGS[WORKLOAD]["seed"], device="cuda:%d" % local_rank)
            ms, res, _ = bench_layout(ctx, torch, pop, min(args.steps, 10), 3, flush, barrier)
            ctx.destroy()
            del ctx
            torch.cuda.empty_cache()
            n_out = int(res["live"].sum())
            nbytes = RECORD_BYTES[main] * (n_tracks + n_out)
            if physics == 2:
                nbytes += 12 * (n_epm + int(res["live"][0]) + int(res["live"][1]))
            t = float(np.mean(ms))
            blk = {"ms_per_step": t, "ms_min": float(np.min(ms)), "track_steps_per_s": n_tracks / (t * 1e-3),
                   "algorithmic_bytes_per_launch": nbytes, "roofline_frac": nbytes / (t * 1e-3) / 1e9 / peak,
                   "vs_physics0_time": t / m["ms_per_step"]}
            if not args.no_cpu:
                _, dt, r = oracle_single_step(pop, n_tracks, want_tracks=True, physics=physics)
                par = full_size_parity(res, r)
                blk.update(counts_bit_exact=par["counts_bit_exact"], tracks_with_another_fate=par["tracks_with_another_fate"],
                           tracks_with_any_word_differing=par["tracks_with_any_word_differing"], cpu_seconds=dt)
                del r
            out["single_step_physics"]["physics%d" % physics] = blk
            del res
    del pop
    torch.cuda.empty_cache()
    if world == 1:
        if "showers" in args.extras:
            out["showers"] = {}
            for name in ("full", "heavy") if "heavy" in args.extras else ("full",):
                # the oracle needs ~80 s for config 5: timed (and its counts compared) only under --extras heavy_cpu;
                # tests/test_gpu_parity.py test_heavy_showers_at_full_size_match_the_oracle holds that parity
                out["showers"][name] = showers(args, name, layout=main, scheme="dense", steps=3, warmup=1,
                                               with_cpu=not args.no_cpu and (name != "heavy" or "heavy_cpu" in args.extras))
            # config 2 under the extended rule set (DESIGN.md rules X36-X39: delta rays, Klein-Nishina sampling,
            # annihilation in flight, multiple scattering), against the oracle under the same rules
            out["showers"]["full_physics2"] = showers(args, "full", layout=main, scheme="dense", steps=3, warmup=1,
                                                      with_cpu=not args.no_cpu, physics=2)
            # the paper's default container on the same workloads: sparse single buffer, AoS, with slot
            # recycling (without it config 5 needs ~5.7e7 e- slots, SURVEY.md:583); parity against the
            # oracle result already computed above
            for name in ("full", "heavy") if "heavy" in args.extras else ("full",):
                b = showers(args, name, layout="aos", scheme="sparse", steps=3, warmup=1, with_cpu=False, flags=1)
                ref = out["showers"][name]
                b["same_counts_as_dense"] = bool(b["track_steps"] == ref["track_steps"] and b["iterations"] == ref["iterations"]
                                                 and b["secondaries"] == ref["secondaries"])
                b["edep_layer_rel_diff_to_dense"] = float(np.max(np.abs(np.array(b["edep_layer_MeV"]) - np.array(ref["edep_layer_MeV"]))
                                                                 / np.maximum(np.array(ref["edep_layer_MeV"]), 1e-30)))
                out["showers"][name + "_sparse_recycle"] = b
        if "sweep" in args.extras:
            # per-field read / write counts (configs[3]): instrumented contexts at 50 % occupancy
            out["sweep"] = sweep(args, layouts=("aos", "soa", "aosoa32", "hc16"), steps=5, warmup=3, instr=True, sections=True,
                                 instr_occupancies=(0.5,))
    emit(out)
    if dist is not None:
        dist.destroy_process_group()


def showers(args, name: str, *, layout: str, scheme: str, steps: int, warmup: int, with_cpu: bool, batch: int = 0,
            flags: int = 0, physics: int = 0) -> dict:
    """BASELINE.json configs[0], [1], [4] (tiny / full / heavy): adept_inject + adept_run to completion,
    wall clock around the two calls (host primaries in, tallies out: this IS the end-to-end number).
    These runs are launch-latency bound for most of their iterations, so no roofline
    fraction is claimed for them."""
    import torch
    from paper_2302_08252_b200 import Context
    from workloads import gen_primaries
    c = CONFIGS[name]
    geo, tab = geometry_for(name), tables_for(name, physics)
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    ctx = Context(geo, tab, layout=layout, scheme=scheme, capacity=c["capacity"], seed=c["seed"],
                  batch_primaries=batch, flags=flags)
    times, res = [], None
    for it in range(warmup + steps):
        ctx.reset()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.inject(prim)                      # host primaries -> device (H2D inside the timed region)
        res = ctx.run()                       # returns the tallies (D2H inside the timed region)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    ctx.destroy()
    del ctx
    torch.cuda.empty_cache()
    n_steps = int(res["steps"].sum())
    t = float(np.mean(times))
    out = {"value": n_steps / t, "unit": "track-steps/s", "ms_per_run": 1e3 * t, "ms_min": 1e3 * float(np.min(times)),
           "runs": steps, "warmup_runs": warmup,
           "workload": "%s showers (BASELINE.json): %d x %g MeV e-, %d layers, adept_inject + adept_run to "
                       "completion, wall clock around the two calls" % (name, c["n_primaries"], c["e_primary"], c["n_layers"]),
           "layout": layout, "scheme": scheme, "capacity_per_kind": c["capacity"], "batch_primaries": batch,
           "slot_recycling": bool(flags & 1), "physics": physics,
           "showers_per_s": c["n_primaries"] / t, "track_steps": n_steps, "iterations": int(res["iterations"]),
           "us_per_iteration": 1e6 * t / max(1, int(res["iterations"])),
           "gpu_launches_per_run": int(res["iterations"]),
           "secondaries": [int(x) for x in res["secondaries"]], "slots_used": [int(x) for x in res["slots_used"]],
           "edep_layer_MeV": [float(x) for x in res["edep_layer"]],
           "energy_balance_rel": float((res["edep_slab"].sum() + res["e_escaped"]) / res["e_injected"] - 1.0),
           "h2d_bytes_per_run": 32 * c["n_primaries"], "d2h_bytes_per_run": 512 + 8 * (2 * c["n_layers"] + 1 + 12)}
    if with_cpu:                                           # heavy: the oracle needs ~80 s
        from oracle import Oracle
        o = Oracle(geo, tab, seed=c["seed"])
        o.inject(prim)
        t0 = time.perf_counter()
        o.run()
        dt = time.perf_counter() - t0
        r = o.result()
        o.close()
        out["cpu_baseline"] = {"value": int(r["steps"].sum()) / dt, "unit": "track-steps/s", "cores": 1,
                               "host_cores": host_cores(), "kind": "oracle", "sample": "the whole %s workload" % name,
                               "seconds": dt}
        keys = ("steps", "secondaries", "killed", "escaped_n")
        out["parity_full_size"] = {
            "counts_bit_exact": bool(all((res[k] == r[k]).all() for k in keys) and res["iterations"] == r["iterations"]),
            "edep_layer_rel_err": float(np.max(np.abs(res["edep_layer"] - r["edep_layer"]) / np.maximum(r["edep_layer"], 1e-30))),
            "e_escaped_rel_err": float(abs(res["e_escaped"] - r["e_escaped"]) / max(r["e_escaped"], 1e-30))}
    return out


def sharded_showers(args, name, rank, world, local_rank, dist, max_over_ranks, reduce_on_cpu=False) -> dict:
    """N > 1: the primaries of `name` split over the ranks, one context per GPU, one
    all-reduce of the tallies at the end (paper_2302_08252_b200/sharding.py).  Strong scaling: the
    total work is fixed."""
    import torch
    from paper_2302_08252_b200 import Context
    from paper_2302_08252_b200.sharding import run_sharded
    from workloads import gen_primaries
    c = CONFIGS[name]
    prim = gen_primaries(c["n_primaries"], c["e_primary"])
    ctx = Context(geometry_for(name), tables_for(name), layout="aosoa32", scheme="dense", capacity=c["capacity"],
                  seed=c["seed"], device="cuda:%d" % local_rank)
    times, res = [], None
    for it in range(1 + 3):
        ctx.reset()
        torch.cuda.synchronize()
        dist.barrier()
        t0 = time.perf_counter()
        res = run_sharded(ctx, prim, rank, world, device="cpu" if reduce_on_cpu else None)
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0)
        if it > 0:
            times.append(dt)
    ctx.destroy()
    n_steps = int(res["steps"].sum())
    t = float(np.mean(times))
    return {"value": n_steps / t, "unit": "track-steps/s", "ms_per_run": 1e3 * t, "scaling": "strong",
            "workload": "%s showers, primaries sharded over %d ranks, one all-reduce of the tallies" % (name, world),
            "track_steps": n_steps, "iterations": int(res["iterations"]), "showers_per_s": c["n_primaries"] / t}


# algorithmic bytes per track-step of one cell of the sweep.  Dense: every record is
# read once and every output record (survivor or secondary) written once.  Sparse: per input track one
# slot-list entry and the record (AoS: its two sectors; SoA family: its 14 words -- the sector
# amplification of scattered slots comes on top and is what the paper's finding is about); per
# survivor the record's dirty bytes (SPARSE_DIRTY_BYTES) and one slot-list entry; per secondary a whole
# record and one slot-list entry.
# Bytes of a record the move half of a step must write back in place (sparse scheme): AoS rewrites
# its two sectors; SoA16 its vectors with a changed word (all four for a photon); HC16 its two hot
# vectors; the word-by-word layouts the 7-8 words a step assigns (pos, nial of the kind, step, ekin / vol).
SPARSE_DIRTY_BYTES = {"aos": 64, "soa16": 56, "hc16": 32}


def sweep_bytes(scheme: str, layout: str, n_in: int, n_surv: int, n_sec: int) -> int:
    rec = RECORD_BYTES[layout]
    if scheme == "dense":
        return rec * (n_in + n_surv + n_sec)
    return n_in * (4 + rec) + n_surv * (SPARSE_DIRTY_BYTES.get(layout, 32) + 4) + n_sec * (rec + 4)


SECTION_NAMES = ("other", "load", "move", "interact", "alloc", "store")


def sweep(args, *, layouts, steps, warmup, instr, sections, occupancies=None, schemes=("dense", "sparse"),
          instr_occupancies=None) -> dict:
    """BASELINE.json configs[3]: 4 Mi slots per kind, occupancy 10..90 %, both schemes x layouts.  Per
    cell: time of one adept_step (CUDA events, state restored and L2 flushed between repetitions) with
    its roofline fraction; the share of that time spent in slot allocation / compaction (rows A9, A10;
    section clocks of the timing variant of the library, include/adept.h) -- the step does both inside
    one kernel, so "step plus allocation/compaction time" is one time and its split; and, with
    `instr`, the per-field read/write counts and slots / 128-byte lines touched
     from an instrumented context of the same population."""
    import torch
    from paper_2302_08252_b200 import Context, FIELD_NAMES
    from workloads import gen_sweep
    c = CONFIGS["sweep"]
    geo, tab = geometry_for("sweep"), tables_for("sweep")
    span, cap = c["span"], c["span"] + c["reserve"]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    peak, peak_src = measured_peak()
    cells = []
    for occ in (occupancies or c["occupancies"]):
        pop = gen_sweep(occ)
        n_live = sum(p["tracks"].shape[0] for p in pop)
        for scheme in schemes:
            for layout in layouts:
                cell = {"occupancy": occ, "scheme": scheme, "layout": layout, "tracks": n_live}
                variants = [("time", False, None)]
                if sections:
                    variants.append(("sections", False, "timing"))
                if instr and (instr_occupancies is None or occ in instr_occupancies):
                    variants.append(("instr", True, None))
                for what, instrument, variant in variants:
                    ctx = Context(geo, tab, layout=layout, scheme=scheme, capacity=cap, seed=c["seed"],
                                  instrument=instrument, variant=variant)
                    for k in range(3):
                        ctx.load_tracks(k, pop[k]["tracks"], pop[k]["slots"] if scheme == "sparse" else None)
                    torch.cuda.synchronize()
                    if what == "time":
                        pristine = ctx.snapshot()
                        ms = []
                        for it in range(warmup + steps):
                            ctx.rewind(pristine)
                            flush.zero_()
                            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                            e0.record(ctx.stream)
                            ctx.step(sync=False)
                            e1.record(ctx.stream)
                            torch.cuda.synchronize()
                            if it >= warmup:
                                ms.append(e0.elapsed_time(e1))
                        res = ctx.result()
                        del pristine
                        t = float(np.mean(ms))
                        n_sec = int(res["secondaries"].sum())
                        n_surv = int(res["live"].sum()) - n_sec
                        nbytes = sweep_bytes(scheme, layout, n_live, n_surv, n_sec)
                        traffic, traffic_src = ncu_traffic("sweep_%g" % occ, layout, scheme)
                        cell.update(ms_per_step=t, ms_min=float(np.min(ms)), track_steps_per_s=n_live / (t * 1e-3),
                                    secondaries=[int(x) for x in res["secondaries"]],
                                    slots_used=[int(x) for x in res["slots_used"]],
                                    algorithmic_bytes=nbytes,
                                    roofline={"bound": "hbm", "achieved": nbytes / (t * 1e-3) / 1e9, "peak": peak,
                                              "unit": "GB/s", "frac": nbytes / (t * 1e-3) / 1e9 / peak,
                                              "traffic": traffic, "traffic_source": traffic_src})
                    elif what == "sections":
                        ctx.step()
                        cyc = ctx.read_sections().astype(np.float64)[:len(SECTION_NAMES)]
                        share = cyc / max(1.0, cyc.sum())
                        cell["section_share"] = {n: float(v) for n, v in zip(SECTION_NAMES, share)}
                        cell["alloc_compaction_ms"] = float((share[4] + share[5]) * cell["ms_per_step"])
                        cell["alloc_ms"] = float(share[4] * cell["ms_per_step"])
                        cell["store_ms"] = float(share[5] * cell["ms_per_step"])
                    else:
                        ctx.step()
                        cnt = ctx.read_counters()
                        rw = cnt["field_rw"].sum(axis=0)                    # over kinds -> [14][2]
                        cell.update(field_reads={n: int(v) for n, v in zip(FIELD_NAMES, rw[:, 0])},
                                    field_writes={n: int(v) for n, v in zip(FIELD_NAMES, rw[:, 1])},
                                    lines_touched=int((cnt["lines"] > 0).sum()),
                                    slots_touched=int((cnt["slots"] > 0).sum()),
                                    bytes_touched_per_track_step=128.0 * float((cnt["lines"] > 0).sum()) / n_live)
                        # the same step's traffic counted in 128-byte lines touched (SURVEY.md §8(d) states the sparse
                        # SoA figure this way) beside the method's own bytes: what sector amplification adds
                        cell["line_bytes"] = 128 * int((cnt["lines"] > 0).sum())
                        cell["line_bytes_over_algorithmic"] = cell["line_bytes"] / max(1, cell["algorithmic_bytes"])
                        cell["roofline"]["frac_line_bytes"] = cell["line_bytes"] / (cell["ms_per_step"] * 1e-3) / 1e9 / peak
                    ctx.destroy()
                    del ctx
                    torch.cuda.empty_cache()
                cells.append(cell)
                # progress, as plain text: the driver takes the LAST JSON-parsable line of the run for the result line
                sys.stderr.write("sweep cell: occupancy %g %s %s  %.4f ms/step  alloc+compaction %s ms  touched %s B/track-step\n"
                                 % (occ, scheme, layout, cell["ms_per_step"], cell.get("alloc_compaction_ms"),
                                    cell.get("bytes_touched_per_track_step")))
        del pop
    best = max(cells, key=lambda x: x["track_steps_per_s"])
    return {"workload": "buffer-scheme sweep (BASELINE.json configs[3]): %d slots per kind, 5 %% of live tracks "
                        "spawn one secondary; one adept_step per cell" % span,
            "peak_source": peak_src,
            "sections": "share of per-warp cycles per kernel section from libadept_b200_timing.so (section clocks), "
                        "applied to the cell's ms_per_step; alloc = rows A9 (ballots, arrival word, reservation, "
                        "group barrier), store = row A10 (record and slot-list writes)" if sections else None,
            "best": {k: best[k] for k in ("occupancy", "scheme", "layout", "ms_per_step", "track_steps_per_s")},
            "cells": cells}


def run_showers_cli(args, name: str):
    """--workload tiny|full|heavy: the shower block as a contract line of its own."""
    layout = "aosoa32" if args.layout == "all" else args.layout
    sampler = ClockSampler(0)
    sampler.start()
    b = showers(args, name, layout=layout, scheme=args.scheme, steps=args.steps, warmup=args.warmup,
                with_cpu=not args.no_cpu, batch=args.batch, flags=1 if args.recycle else 0, physics=args.physics)
    clocks = sampler.stop()
    out = {"metric": "track-steps/sec", "value": b["value"], "unit": "track-steps/s", "n_gpus": 1,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": b["ms_per_run"], "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": b["workload"], "layout": layout, "scheme": args.scheme,
                      "capacity_per_kind": b["capacity_per_kind"], "batch_primaries": args.batch},
           "clocks": clocks, "gpu_launches": b["gpu_launches_per_run"],
           "e2e": {"value": b["value"], "unit": "track-steps/s", "h2d_bytes_per_step": b["h2d_bytes_per_run"],
                   "d2h_bytes_per_step": b["d2h_bytes_per_run"],
                   "what": "same measurement: the timed region is the public API with host buffers"},
           "roofline": None}
    out.update({k: v for k, v in b.items() if k not in ("value", "unit", "workload")})
    print(json.dumps(out))


def run_sweep_cli(args):
    layouts = ("aos", "soa", "aosoa32", "aosoa64", "soa16", "hc16") if args.layout == "all" else (args.layout,)
    sw = sweep(args, layouts=layouts, steps=args.steps, warmup=args.warmup, instr=not args.no_instr,
               sections=not args.no_sections,
               occupancies=None if args.occupancy is None else (args.occupancy,),
               schemes=("dense", "sparse") if args.scheme is None else (args.scheme,))
    best = sw["best"]
    out = {"metric": "track-steps/sec", "value": best["track_steps_per_s"], "unit": "track-steps/s",
           "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": best["ms_per_step"],
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": sw["workload"] + "; value = best cell", "layout": best["layout"],
                      "scheme": best["scheme"], "occupancy": best["occupancy"]},
           "gpu_launches": args.steps, "roofline": None}
    out.update({k: sw[k] for k in ("peak_source", "sections", "cells")})
    print(json.dumps(out))


def relaunch_as_ranks(n: int) -> int:
    """`python bench.py --gpus N` outside torchrun: run the same command line as N ranks of one node."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--layout", default="all", choices=["soa", "aosoa32", "aosoa64", "soa16", "aos", "aosoa16", "aosoa128", "hc16", "aosoa8", "all"])
    ap.add_argument("--tracks", type=int, default=CONFIGS[WORKLOAD]["n_tracks"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline legs")
    ap.add_argument("--extras", default=None,
                    help="comma list of what the default line carries beside the headline: showers, heavy, sweep, physics "
                         "(default: all four at the full population, none otherwise); heavy_cpu = also time the oracle on "
                         "config 5 (~80 s); 'none' = headline only")
    ap.add_argument("--workload", default="single_step", choices=["single_step", "tiny", "full", "heavy", "sweep"],
                    help="single_step = the headline (BASELINE.json configs[2]); the others as a line of their own")
    ap.add_argument("--scheme", default=None, choices=["dense", "sparse"],
                    help="shower workloads: container (default dense); sweep: only this scheme (default both)")
    ap.add_argument("--occupancy", type=float, default=None, help="sweep: only this occupancy (default 0.1 .. 0.9)")
    ap.add_argument("--no-instr", action="store_true", help="sweep: skip the instrumented (counting) contexts")
    ap.add_argument("--no-sections", action="store_true", help="sweep: skip the section-clock contexts")
    ap.add_argument("--batch", type=int, default=0, help="shower workloads: batch_primaries (0 = all at once)")
    ap.add_argument("--recycle", action="store_true", help="shower workloads, sparse scheme: recycle freed slots")
    ap.add_argument("--physics", type=int, default=0, choices=[0, 1, 2], help="shower workloads: adept_tables.physics")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        sys.exit(relaunch_as_ranks(args.gpus))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and rank == 0:
        sys.stderr.write("bench.py: --gpus %d but %d rank(s) were launched; reporting n_gpus = %d\n" % (args.gpus, world, world))
    if args.extras is None:
        args.extras = "showers,heavy,sweep,physics" if args.tracks == CONFIGS[WORKLOAD]["n_tracks"] else "none"
    args.extras = set(x for x in args.extras.split(",") if x and x != "none")
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.workload in ("tiny", "full", "heavy"):
        if rank == 0:
            args.scheme = args.scheme or "dense"
            run_showers_cli(args, args.workload)
        return
    if args.workload == "sweep":
        if rank == 0:
            run_sweep_cli(args)
        return
    run_gpu(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
