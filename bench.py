#!/usr/bin/env python
"""bench.py -- events/s of the whole hot path (S1 layout -> S2..S6 tracking -> S7 ghost-killer MLP -> S8..S10 vertexing)
on BASELINE.json configs[4]: 100 000 synthetic Run-3-shaped events (cfg-1 generator, seed 4), device resident,
processed as 10 sub-batches of 10 000 events on two CUDA streams.  One JSON line on stdout (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W]                 # this library (CUDA, sm_100a)
    python bench.py --impl reference [--steps K] [--warmup W]           # the fp64 CPU oracle on the host cores
    torchrun --nproc-per-node N ... bench.py --gpus N ...               # one rank per GPU, weak scaling, no collective
                                                                        # on the data path (events are independent)

A step = one pass of the whole path over all sub-batches.  `value` = events of all ranks / (device time of K steps,
max over ranks).  `e2e` = the same through ds_process_host with pinned HOST buffers (H2D of every input and D2H of all
tracks and vertices inside the timed region).  `roofline` = the kernel with the largest share of the step: its
algorithmic bytes / its CUDA-event time measured in the timed region / the measured HBM peak.
`cpu_baseline` = oracle/ as it stands on a bounded sample of the same events, same box.
"""
from __future__ import annotations

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

METRIC = "events_per_s_downstream_mlp_vertexing"
UNIT = "events/s"
CFG = 4


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ---- inputs --------------------------------------------------------------------------------------------------------------
def generate_subbatches(rank: int, n_sub: int, sub_events: int, workers: int):
    """Sub-batch i of rank r = RNG blocks [r*n_sub*B + i*B, ... + B) of cfg4 (B = blocks per sub-batch)."""
    import gen
    from gen import constants as C
    from paper_2503_13092_b200 import shard
    bps = -(-sub_events // C.BLOCK_EVENTS)
    b0, _ = shard.block_range(rank, n_sub * bps)
    out = []
    for i in range(n_sub):
        d = gen.generate(CFG, n_events=sub_events, first_block=b0 + i * bps, workers=workers)
        d.pop("truth", None)
        out.append(d)
    return out


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic():
    """dram bytes per launch per kernel from the committed ncu --set full capture, if there is one."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f)
    return {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md, clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, smax, reasons, power = [], [], set(), []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---- algorithmic bytes -------------------------------------------------------------
def algorithmic_bytes(n_events, n_hits, n_seeds, n_found, n_keep, n_vtx):
    return {
        "k_layout": 52 * n_hits + 57 * 4 * n_events,                       # read 24 B/hit, write 24 + 4 B/hit, bin table
        "k_track": 20 * n_hits + 28 * n_seeds + 52 * n_seeds + 16 * n_found,  # sorted hit fields once, seeds in, tracks out, 4 ids
        "k_mlp": 12 * n_seeds + 32 * n_found,                              # found in, score + keep out; 8 features of found tracks
        "k_vertex_count": 28 * n_keep + 8 * n_seeds + 4 * n_events,
        "k_vertex_scan": 16 * n_events,
        "k_vertex_write": 28 * n_keep + 40 * n_vtx,
        # S1..S6 in one launch: the S1 and S2..S6 figures of SURVEY 8d together (what the unfused algorithm moves)
        "k_event": 52 * n_hits + 57 * 4 * n_events + 20 * n_hits + 28 * n_seeds + 52 * n_seeds + 16 * n_found,
        "k_clone": 28 * n_seeds,                                           # hit[4], chi2, nhits, found of every slot
        "k_lines": (24 + 32 + 20) * n_vtx,                                 # vertex record, 2 x 4 track values, 4 scores + bits
    }


# ---- the oracle arm --------------------------------------------------------------------------------------------------------
def oracle_events_per_s(d, n_events, n_threads=0):
    """Time oracle.reconstruct + oracle.vertex on the first n_events events of d (n_threads = 0: all host cores, OpenMP)."""
    import gen
    from gen import constants as C
    from oracle import ds_oracle as O
    sub = gen.take_events(d, n_events)
    mlp = O.Mlp(gen.mlp_weights(0))
    t0 = time.perf_counter()
    r = O.reconstruct(sub["hits"], sub["hit_offsets"], sub["seeds"], sub["seed_offsets"], C.GEOMETRY, C.PARAMS, mlp, n_threads=n_threads)
    v = O.vertex(r, sub["seed_offsets"], C.GEOMETRY, C.PARAMS, n_threads=n_threads)
    dt = time.perf_counter() - t0
    return n_events / dt, dt, (n_threads or O.max_threads()), int(r["found"].sum()), v["n"]


def sized_sample(d, target_s, cap):
    rate, _, _, _, _ = oracle_events_per_s(d, min(200, cap))
    return int(max(100, min(cap, rate * target_s)))


def run_reference(args, rank):
    """--impl reference: there is no reference implementation for this paper; the arm is the fp64 CPU oracle."""
    if rank != 0:
        return
    import gen
    from gen import constants as C
    if args.magnet_polarity != 0.0:
        C.PARAMS = dict(C.PARAMS, magnet_polarity=args.magnet_polarity)
    if args.dv1:
        C.PARAMS = dict(C.PARAMS, dv1=1)
    d = gen.generate(CFG, n_events=args.subbatch, workers=min(8, os.cpu_count() or 1))
    per_step = min(10.0, 150.0 / max(1, args.steps + args.warmup))
    n = sized_sample(d, per_step, args.subbatch)
    for _ in range(args.warmup):
        oracle_events_per_s(d, n)
    t0 = time.perf_counter()
    cores = 1
    for _ in range(args.steps):
        _, _, cores, _, _ = oracle_events_per_s(d, n)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = f"first {n} events of cfg4 sub-batch 0 per step (oracle/ds_oracle.c, fp64, OpenMP over events)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE configs[4]: cfg-1 generator, seed 4 (bounded sample)", "events_per_step": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


# ---- our arm -------------------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=100000, help="events per GPU (BASELINE configs[4]: 100 000)")
    ap.add_argument("--subbatch", type=int, default=10000)
    ap.add_argument("--streams", type=int, default=2)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cfg", type=int, default=4, choices=[1, 2, 3, 4],
                    help="BASELINE configs[k] generator; 4 = the metric's workload.  3 (with --events 2000 --subbatch 2000): the "
                         "vertexing stress, reported with the ALU fraction of the vertex kernels (SURVEY 8d)")
    ap.add_argument("--lines", action="store_true",
                    help="also run the four HLT1 line NNs on the vertices (SURVEY 8f N4, P:277-P:285) in our arm")
    ap.add_argument("--dv1", action="store_true",
                    help="Dv1 triplet search instead of the Dv0 first window (SURVEY 8f N2, P:107-P:111) in both arms")
    ap.add_argument("--clone-min-shared", type=int, default=0,
                    help="3: clone killing across seeds between S6 and S7 (SURVEY 8f N3, P:115); 0 = BASELINE configs")
    ap.add_argument("--mlp", default="cfg", choices=["cfg", "paper"],
                    help="paper: the ghost killer is the paper's 8 -> 14 -> 1 network (P:121, SURVEY 8f N5) in our arm")
    ap.add_argument("--mlp-fast-math", action="store_true",
                    help="ghost-killer sigmoid by __expf / __fdividef as in the paper (P:157); the line then carries `mlp_variant` "
                         "with the score differences against the IEEE path")
    ap.add_argument("--no-legs", action="store_true", help="skip the short cfg3 / cfg2 legs that follow the cfg4 timing")
    ap.add_argument("--magnet-polarity", type=float, default=0.0,
                    help="+1 / -1: curved-track vertexing (SURVEY 8f N1, P:255-P:269) in both arms; 0 = BASELINE configs")
    args = ap.parse_args()
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    global CFG
    CFG = args.cfg
    if args.impl == "reference":
        return run_reference(args, rank)
    if args.warmup < 3:
        log("note: the timing rules ask for >= 3 warm-up steps")

    from gen import constants as C
    import gen
    if args.magnet_polarity != 0.0:   # both arms (the oracle legs read C.PARAMS) vertex with the parabolas of Eq. 4
        C.PARAMS = dict(C.PARAMS, magnet_polarity=args.magnet_polarity)
    if args.dv1:
        C.PARAMS = dict(C.PARAMS, dv1=1)
    if args.clone_min_shared:         # our arm only: the timed oracle legs have no clone-killing step
        C.PARAMS = dict(C.PARAMS, clone_min_shared=args.clone_min_shared)
    n_sub = max(1, args.events // args.subbatch)
    workers = max(1, min(32, (os.cpu_count() or 1) // max(1, world)))
    t0 = time.time()
    subs = generate_subbatches(rank, n_sub, args.subbatch, workers)      # before CUDA is touched: the pool forks
    log(f"[rank {rank}] generated {n_sub} x {args.subbatch} events in {time.time() - t0:.1f} s ({workers} workers)")

    import torch
    import torch.distributed as dist
    import paper_2503_13092_b200 as pk
    from paper_2503_13092_b200 import shard
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- pinned host copies (e2e inputs) and device-resident copies (kernel-path inputs) --------------------------------
    mlp_w = gen.mlp_weights(0)
    # max_event_hits_hint = the largest event of the workload (sizes the kernels' per-event staging buffers)
    max_event_hits = max(int(np.diff(d["hit_offsets"]).max()) for d in subs)
    params = dict(C.PARAMS, max_event_hits_hint=max_event_hits)
    ds = pk.Downstream(C.GEOMETRY, mlp_w, params, device=local)
    if args.mlp == "paper":
        ds.upload_mlp_single(gen.mlp_single_weights(0))
    host, devd = [], []
    for d in subs:
        hp = dict(hits={k: torch.from_numpy(v).pin_memory() for k, v in d["hits"].items()},
                  seeds={k: torch.from_numpy(v).pin_memory() for k, v in d["seeds"].items()},
                  hit_offsets=torch.from_numpy(d["hit_offsets"]).pin_memory(),
                  seed_offsets=torch.from_numpy(d["seed_offsets"]).pin_memory(), n_events=d["n_events"])
        host.append(hp)
        devd.append(dict(hits={k: v.to(dev, non_blocking=True) for k, v in hp["hits"].items()},
                         seeds={k: v.to(dev, non_blocking=True) for k, v in hp["seeds"].items()},
                         hit_offsets=hp["hit_offsets"].to(dev, non_blocking=True),
                         seed_offsets=hp["seed_offsets"].to(dev, non_blocking=True), n_events=d["n_events"]))
    n_hits = [int(d["hit_offsets"][-1]) for d in subs]
    n_seeds = [int(d["seed_offsets"][-1]) for d in subs]
    first_sub = subs[0]
    del subs
    torch.cuda.synchronize()
    n_streams = max(1, args.streams)
    streams = [torch.cuda.Stream(device=dev) for _ in range(n_streams)]
    cap = 1 << 20 if args.cfg != 3 else 1 << 24   # vertex capacity per sub-batch (cfg3: tens of thousands of pairs per event)
    ws = [ds.workspace(args.subbatch, max(n_hits), max(n_seeds)) for _ in range(n_streams)]
    vws = [ds.vertex_workspace(args.subbatch, max(n_seeds)) for _ in range(n_streams)]
    trk = [ds.empty_tracks(n) for n in n_seeds]
    vtx = [ds.empty_vertices(cap, args.subbatch) for _ in range(n_sub)]
    line_out = None
    if args.lines:
        ds.upload_line_nets(gen.line_weights(0))
        line_out = [dict(scores=torch.zeros((cap, 4), dtype=torch.float32, device=dev),
                         bits=torch.zeros(cap, dtype=torch.int32, device=dev)) for _ in range(n_sub)]

    def run_lines(i, s):
        if line_out is not None:
            pk.ds_lines(ds.h, trk[i], vtx[i], cap, args.subbatch, 0.5, line_out[i]["scores"], line_out[i]["bits"], s)

    def step():
        for i, d in enumerate(devd):
            s = streams[i % n_streams]
            ds.reconstruct(d["hits"], d["seeds"], d["hit_offsets"], d["seed_offsets"], out=trk[i], workspace=ws[i % n_streams], stream=s)
            ds.vertex(trk[i], d["seed_offsets"], out=vtx[i], workspace=vws[i % n_streams], stream=s)
            run_lines(i, s)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    n_found = sum(int(t["found"].sum().item()) for t in trk)
    n_keep = sum(int(t["keep"].sum().item()) for t in trk)
    n_vtx = sum(int(v["offsets"][-1].item()) for v in vtx)
    assert all(int(v["overflow"].item()) == 0 for v in vtx), "vertex capacity overflow"

    # ---- timed region: K steps on the two streams, CUDA events on the stream the work is launched from, clocks sampled ----
    main_stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pk.ds_profile_enable(ds.h, True)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    ev0.record(main_stream)
    for s in streams:
        s.wait_stream(main_stream)
    for _ in range(args.steps):
        step()
    for s in streams:
        main_stream.wait_stream(s)
    ev1.record(main_stream)
    barrier()
    clocks = sampler.stop()
    ms_total = shard.max_over_ranks(ev0.elapsed_time(ev1), dev)
    prof2 = pk.ds_profile_read(ds.h)              # per-kernel events of the timed region: kernels of the two streams overlap
    events_rank = args.subbatch * n_sub
    events_all = shard.sum_over_ranks(events_rank, dev)
    value = events_all * args.steps / (ms_total * 1e-3)

    # ---- spread: the same step K more times, each timed on its own (median and best) ---------------------------------
    per_step = []
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(main_stream)
        for s in streams:
            s.wait_stream(main_stream)
        step()
        for s in streams:
            main_stream.wait_stream(s)
        b.record(main_stream)
        torch.cuda.synchronize()
        per_step.append(a.elapsed_time(b))
    pk.ds_profile_read(ds.h)                      # drop the events of these steps
    step_ms = {"median": statistics.median(per_step), "best": min(per_step), "n": len(per_step)}

    # ---- per-kernel pass: the same K steps, same launches, on ONE stream so that a kernel's event pair times that kernel
    #      alone (in the two-stream region above a pair also spans whatever the other stream runs at the same time) ----------
    def step_one_stream():
        for i, d in enumerate(devd):
            ds.reconstruct(d["hits"], d["seeds"], d["hit_offsets"], d["seed_offsets"], out=trk[i], workspace=ws[0], stream=streams[0])
            ds.vertex(trk[i], d["seed_offsets"], out=vtx[i], workspace=vws[0], stream=streams[0])
            run_lines(i, streams[0])

    barrier()
    for _ in range(args.steps):
        step_one_stream()
    barrier()
    prof = pk.ds_profile_read(ds.h)
    pk.ds_profile_enable(ds.h, False)

    # ---- roofline of the dominant kernel --------------------------------------------------------------------------------------
    peak, peak_src = peaks()
    alg = algorithmic_bytes(events_rank, sum(n_hits), sum(n_seeds), n_found, n_keep, n_vtx)     # bytes per step
    traffic = ncu_traffic()
    kernels, launches = {}, sum(n for _, n in prof2.values())
    leftover = ("k_layout", "k_track") if prof.get("k_event", (0, 0))[1] else ()   # with k_event: launches for the events it leaves
    for name, (ms, n) in prof.items():                                                # over -- none in this workload
        if n == 0:
            continue
        per_launch_ms = ms / n
        if name in leftover:
            alg[name] = 0
        bytes_per_launch = alg[name] * args.steps / n
        gbs = bytes_per_launch / (per_launch_ms * 1e-3) / 1e9
        kernels[name] = {"ms_per_launch": per_launch_ms, "ms_per_step": ms / args.steps, "launches_per_step": n / args.steps,
                         "alg_bytes_per_launch": bytes_per_launch, "achieved_gbs": gbs, "frac": gbs / peak,
                         "traffic": traffic.get(name), "ms_per_launch_two_streams": prof2[name][0] / max(1, prof2[name][1])}
        if name in leftover:
            kernels[name].update(traffic=None, note="launch for the events above k_event's staging capacity: none here, its blocks leave at once")
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_step"])
    ksum = sum(k["ms_per_step"] for k in kernels.values())
    # k_event runs S1..S6 in one launch: its algorithmic bytes are the S1 and S2..S6 figures of SURVEY 8d together (what the
    # steps move when each runs as its own HBM-bound kernel); `min_traffic` is what the fused launch has to move at least
    # (every input array once, seeds in, tracks out) and `traffic` what ncu measured it to move
    fused_min = (24 * sum(n_hits) + 28 * sum(n_seeds) + 52 * sum(n_seeds) + 16 * n_found) * args.steps
    if "k_event" in kernels:
        ke = kernels["k_event"]
        ke["covers"] = "S1..S6 (layout, extrapolation, window searches, fits, best candidate)"
        ke["min_traffic_bytes_per_launch"] = fused_min / (ke["launches_per_step"] * args.steps)
        ke["min_traffic_gbs"] = ke["min_traffic_bytes_per_launch"] / (ke["ms_per_launch"] * 1e-3) / 1e9
        ke["min_traffic_frac"] = ke["min_traffic_gbs"] / peak
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dom]["frac"], "traffic": kernels[dom]["traffic"], "peak_source": peak_src,
                "share_of_step": kernels[dom]["ms_per_step"] / ksum,
                "alg_bytes_per_launch": kernels[dom]["alg_bytes_per_launch"],
                "alg_bytes_basis": "SURVEY 8d per-unit figures of the steps the launch covers x the units of one launch (DESIGN.md section 8)",
                "timing": "CUDA events around every launch, one-stream pass of the same K steps right after the timed region"}
    if dom == "k_event":
        roofline.update(covers=kernels[dom]["covers"], min_traffic_frac=kernels[dom]["min_traffic_frac"])
    # the launches of the leftover path are not part of the sum when they are empty
    whole_gbs = sum(alg[k] for k in kernels if not ("k_event" in kernels and k in ("k_layout", "k_track"))) * args.steps / (ms_total * 1e-3) / 1e9
    # the kernel BASELINE north_star sets the 40 % bar on: search + fit (S2..S6) -- k_event, which does them with S1 in one launch
    roofline_search_fit = None
    sf = "k_event" if "k_event" in kernels else ("k_track" if "k_track" in kernels else None)
    if sf:
        kt = kernels[sf]
        roofline_search_fit = {"bound": "hbm", "kernel": sf, "achieved": kt["achieved_gbs"], "peak": peak, "unit": "GB/s",
                               "frac": kt["frac"], "traffic": kt["traffic"], "share_of_step": kt["ms_per_step"] / ksum}
        if sf == "k_event":
            roofline_search_fit.update(covers=kt["covers"], min_traffic_frac=kt["min_traffic_frac"])

    # ---- cfg3: the vertex kernels are bound by plain fp64 arithmetic, not by HBM -----------------------------------
    def vertex_alu_of(kern, trk_list, dev_list, n_pass):
        """fp64 ALU fraction of the vertex kernels: ~130 flop per pair.  The count kernel evaluates every
        opposite-charge pair, the write kernel only the passing ones again."""
        n_pairs = 0
        for t, d in zip(trk_list, dev_list):
            so = d["seed_offsets"].cpu().numpy()
            keep, q = t["keep"].cpu().numpy(), t["qop"].cpu().numpy()
            pos = np.concatenate([[0], np.cumsum((keep == 1) & (q > 0))])
            neg = np.concatenate([[0], np.cumsum((keep == 1) & (q < 0))])
            n_pairs += int(((pos[so[1:]] - pos[so[:-1]]) * (neg[so[1:]] - neg[so[:-1]])).sum())
        peak_tf = pk.ds_measure_dfma_peak(ds.h)
        out = {"bound": "alu", "pairs_per_step": n_pairs, "passing_pairs_per_step": n_pass, "flop_per_pair": 130,
               "unit": "TFLOP/s (fp64)", "peak": peak_tf,
               "peak_source": "measured: ds_measure_dfma_peak (register-resident DFMA loop on every SM)",
               "peak_nominal": 148 * 64 * 2 * (clocks.get("sm_mhz") or 1965.0) * 1e6 / 1e12}
        if "k_vertex_count" in kern:
            ms_c = kern["k_vertex_count"]["ms_per_step"]
            out["count_kernel"] = {"ms_per_step": ms_c, "achieved": 130.0 * n_pairs / (ms_c * 1e-3) / 1e12}
            out["count_kernel"]["frac"] = out["count_kernel"]["achieved"] / peak_tf
        ms = sum(kern[k]["ms_per_step"] for k in ("k_vertex_count", "k_vertex_write") if k in kern)
        flop = 130.0 * (n_pairs + n_pass)
        out.update(ms_per_step=ms, achieved=flop / (ms * 1e-3) / 1e12, frac=flop / (ms * 1e-3) / 1e12 / peak_tf)
        return out

    vertex_alu = vertex_alu_of(kernels, trk, devd, n_vtx) if args.cfg == 3 else None

    # ---- short legs on the other configurations, one stream, per-kernel events (not the metric: evidence for the kernels
    #      whose regime cfg4 does not show -- the vertexing stress cfg3 and the high-occupancy cfg2) ---------------------------
    legs = {}
    if args.cfg == 4 and not args.no_legs and rank == 0:
        for cfg_k, n_ev in ((3, 2000), (2, 1000)):
            dl = gen.generate(cfg_k, n_events=n_ev, workers=workers)
            dl.pop("truth", None)
            mh = int(np.diff(dl["hit_offsets"]).max())
            ds.set_params(dict(params, max_event_hits_hint=mh))
            dd = dict(hits=ds.to_device(dl["hits"]), seeds=ds.to_device(dl["seeds"]),
                      hit_offsets=ds.to_device(dict(h=dl["hit_offsets"]))["h"], seed_offsets=ds.to_device(dict(s=dl["seed_offsets"]))["s"])
            nh_l, ns_l = int(dl["hit_offsets"][-1]), int(dl["seed_offsets"][-1])
            t_l, v_l = ds.empty_tracks(ns_l), ds.empty_vertices(1 << 22, n_ev)
            w_l, vw_l = ds.workspace(n_ev, nh_l, ns_l), ds.vertex_workspace(n_ev, ns_l)

            def leg_step():
                ds.reconstruct(dd["hits"], dd["seeds"], dd["hit_offsets"], dd["seed_offsets"], out=t_l, workspace=w_l, stream=streams[0])
                ds.vertex(t_l, dd["seed_offsets"], out=v_l, workspace=vw_l, stream=streams[0])
            for _ in range(3):
                leg_step()
            torch.cuda.synchronize()
            pk.ds_profile_enable(ds.h, True)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(streams[0])
            for _ in range(args.steps):
                leg_step()
            b.record(streams[0])
            torch.cuda.synchronize()
            pl = pk.ds_profile_read(ds.h)
            pk.ds_profile_enable(ds.h, False)
            assert int(v_l["overflow"].item()) == 0
            nf_l, nk_l, nv_l = int(t_l["found"].sum().item()), int(t_l["keep"].sum().item()), int(v_l["offsets"][-1].item())
            alg_l = algorithmic_bytes(n_ev, nh_l, ns_l, nf_l, nk_l, nv_l)
            kl = {}
            for name, (ms, n) in pl.items():
                if n and pl.get("k_event", (0, 0))[1] and name in ("k_layout", "k_track"):
                    alg_l[name] = 0   # launches for the events k_event leaves over: none
                if n:
                    gbs = alg_l[name] * args.steps / n / (ms / n * 1e-3) / 1e9
                    kl[name] = {"ms_per_launch": ms / n, "ms_per_step": ms / args.steps, "alg_bytes_per_launch": alg_l[name] * args.steps / n,
                                "achieved_gbs": gbs, "frac": gbs / peak}
            ms_l = a.elapsed_time(b) / args.steps
            legs[f"cfg{cfg_k}"] = {"workload": f"BASELINE configs[{cfg_k}], {n_ev} events, one stream", "events": n_ev, "hits": nh_l, "seeds": ns_l,
                                   "tracks_found": nf_l, "tracks_kept": nk_l, "vertices": nv_l, "ms_per_step": ms_l,
                                   "events_per_s": n_ev / (ms_l * 1e-3), "kernels": kl}
            if cfg_k == 3:
                legs["cfg3"]["vertex_alu"] = vertex_alu_of(kl, [t_l], [dd], nv_l)
            del dd, t_l, v_l, w_l, vw_l, dl
        ds.set_params(params)

    # ---- ghost-killer variants: the other arithmetic flavour on the same tracks, k_mlp alone -------------------
    mlp_variant = None
    if args.mlp_fast_math and rank == 0:
        ref_scores = [t["score"].clone() for t in trk]
        ref_keep = [t["keep"].clone() for t in trk]
        res = {}
        for fast in (0, 1):
            ds.set_params(dict(params, mlp_fast_math=fast))
            pk.ds_profile_enable(ds.h, True)
            for _ in range(args.steps):
                for i, d in enumerate(devd):
                    ds.ghost_killer(d["seeds"], trk[i], stream=streams[0])
            torch.cuda.synchronize()
            ms, n = pk.ds_profile_read(ds.h)["k_mlp"]
            pk.ds_profile_enable(ds.h, False)
            res[fast] = ms / n
        dmax = max(float((t["score"] - r).abs().max().item()) for t, r in zip(trk, ref_scores))
        flips = sum(int((t["keep"] != r).sum().item()) for t, r in zip(trk, ref_keep))
        mlp_variant = {"network": "8-14-1 (P:121)" if args.mlp == "paper" else "8-32-16-1 (BASELINE cfg0)",
                       "k_mlp_ms_per_launch_ieee": res[0], "k_mlp_ms_per_launch_fast_math": res[1],
                       "max_abs_score_difference": dmax, "keep_decisions_flipped": flips, "tracks": n_found,
                       "intrinsics": "__expf, __fdividef (P:157); no fp64 re-evaluation next to the threshold"}
        ds.set_params(params)
        for i, d in enumerate(devd):
            ds.ghost_killer(d["seeds"], trk[i], stream=streams[0])
        torch.cuda.synchronize()

    # ---- end to end: pinned host buffers in, pinned host buffers out, through ds_process_host ----------------------------
    e2e = None
    if not args.no_e2e:
        handles = [pk.Downstream(C.GEOMETRY, mlp_w, params, device=local) for _ in range(n_streams)]
        vcap = 1 << 18
        out_t = [pk.host_tracks(max(n_seeds), pinned=True) for _ in range(n_streams)]
        out_v = [pk.host_vertices(vcap, args.subbatch, pinned=True) for _ in range(n_streams)]
        totals = [0] * n_streams

        def worker(k):
            torch.cuda.set_device(local)
            tot = 0
            for i in range(k, n_sub, n_streams):
                h = host[i]
                ot = {kk: (v[: n_seeds[i]] if kk != "hit" else v[: n_seeds[i]]) for kk, v in out_t[k].items()}
                tot += handles[k].process_host(h["hits"], h["seeds"], h["hit_offsets"], h["seed_offsets"], ot, out_v[k], vcap,
                                               stream=streams[k])
            totals[k] = tot

        def e2e_step():
            th = [threading.Thread(target=worker, args=(k,)) for k in range(n_streams)]
            for t in th:
                t.start()
            for t in th:
                t.join()

        e2e_step()                                              # warm-up (grows the handles' arenas)
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(main_stream)
        for _ in range(max(1, args.e2e_steps)):
            e2e_step()
        b.record(main_stream)
        barrier()
        e2e_ms = shard.max_over_ranks(a.elapsed_time(b), dev)
        assert sum(totals) == n_vtx, "e2e path and device path disagree on the number of vertices"
        h2d = 24 * sum(n_hits) + 24 * sum(n_seeds) + 2 * 4 * (events_rank + n_sub)
        d2h = 56 * sum(n_seeds) + 40 * n_vtx + (4 + 8) * events_rank + 12 * n_sub
        e2e = {"value": events_all * max(1, args.e2e_steps) / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": max(1, args.e2e_steps), "ms_per_step": e2e_ms / max(1, args.e2e_steps),
               "api": "ds_process_host, pinned host buffers, one handle + stream per thread"}
        for h in handles:
            h.close()

    # ---- the oracle beside it (rank 0, N = 1): all host cores and one thread, on the first cfg4 sub-batch and on cfg1
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import ds_oracle as O
        ncores = O.max_threads()
        n = sized_sample(first_sub, 12.0, args.subbatch)
        v, dt, cores, _, _ = oracle_events_per_s(first_sub, n, ncores)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"first {n} events of cfg{CFG} sub-batch 0 (oracle/ds_oracle.c, fp64, OpenMP over events)"}
        legs_cpu = {}
        n1 = int(max(50, min(n, v / max(1, ncores) * 5.0)))
        v1, dt1, _, _, _ = oracle_events_per_s(first_sub, n1, 1)
        legs_cpu[f"cfg{CFG}_1_thread"] = {"value": v1, "cores": 1, "seconds": dt1, "sample": f"first {n1} events of cfg{CFG} sub-batch 0"}
        d1 = gen.generate(1, n_events=1000, workers=workers)
        va, dta, _, _, _ = oracle_events_per_s(d1, 1000, ncores)
        legs_cpu["cfg1_all_cores"] = {"value": va, "cores": ncores, "seconds": dta, "sample": "BASELINE configs[1], 1000 events"}
        n11 = int(max(50, min(1000, va / max(1, ncores) * 4.0)))
        vb, dtb, _, _, _ = oracle_events_per_s(d1, n11, 1)
        legs_cpu["cfg1_1_thread"] = {"value": vb, "cores": 1, "seconds": dtb, "sample": f"first {n11} events of BASELINE configs[1]"}
        cpu["legs"] = legs_cpu

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "step_ms": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": ("BASELINE configs[4]: cfg-1 generator, seed 4, device-resident SoA" if CFG == 4 else
                                    f"BASELINE configs[{CFG}] generator, device-resident SoA (not the metric's workload)"),
                       "events_per_gpu": events_rank,
                       "subbatches": n_sub, "events_per_subbatch": args.subbatch, "cuda_streams": n_streams,
                       "hits": sum(n_hits), "seeds": sum(n_seeds), "tracks_found": n_found, "tracks_kept": n_keep, "vertices": n_vtx,
                       "l2": "inputs larger than L2 (each sub-batch reads ~0.76 GB; 7.6 GB per step)",
                       "magnet_polarity": args.magnet_polarity, "clone_min_shared": args.clone_min_shared, "dv1": bool(args.dv1), "lines": bool(args.lines), "mlp": args.mlp,
                       "parallelism": f"dp{world} (events sharded, no data-path collective)"},
            "roofline": roofline, "roofline_search_fit": roofline_search_fit, "legs": legs, "mlp_variant": mlp_variant,
            "whole_path_gbs": whole_gbs, "whole_path_frac": whole_gbs / peak, "kernels": kernels,
            "vertex_alu": vertex_alu, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        }), flush=True)
    ds.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
