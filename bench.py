#!/usr/bin/env python
"""bench.py — measures BASELINE.json's metric for the DKD + descriptor-sampling hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

One JSON line on stdout (rank 0).  A "step" is ONE pass of the whole hot path (NMS -> top-k ->
refinement -> descriptor gather) over one 752x480 stereo pair of config c2
(BASELINE.json configs[1], the configuration the metric "us per 752x480 stereo pair" is quoted on),
through the C-ABI (`dkd_extract`, one cached CUDA-graph launch).  Per rank:

  * value / ms_per_step : the MEDIAN over --blocks (50) back-to-back blocks of exactly K steps each on inputs
                          resident in HBM, CUDA events on the launching stream (one between blocks), barrier +
                          synchronize on both sides of the series, max over ranks; min / median / p95 in
                          `value_blocks`.  Cold inputs: the steps rotate through R distinct seeded input sets
                          whose touched bytes exceed L2.
  * e2e                 : the same K steps through `dkd_extract_host` with pinned HOST buffers, everything inside
                          the timed region: the score maps are copied host->device, the descriptor corner rows
                          are read in place from the pinned map over PCIe (counted as h2d bytes), and the kernels
                          store every output into the pinned host tensors (d2h bytes); synchronised per step.
  * fresh_buffers       : the same steps with output buffers the cached graph has not seen (kernel-node update path).
  * batch64 / roofline  : config c5 (B=64 1080p, BASELINE.json configs[4]); whole-path frames/s,
                          keypoints/s, credited GB/s, and the dominant kernel's duration measured with
                          CUDA events (library measurement mode) against MEASURED_PEAKS.json.
  * variants_c5         : c5 with the heat x reliability and validity-mask variants (NMS credited 8 B / 9 B per pixel).
  * match / retrieval   : the consumers of the descriptors: tcgen05 matching (tensor roofline; also with
                          the mutual check) and the keyframe-database cosine scan (HBM roofline); the f4 kernels per call;
                          `match.frontend_frame_us`: the composed chain extract(B=4) -> match(P=2) -> stereo validation
                          captured in one caller graph, at keypoint caps 256 and 1024.
  * other_configs       : c1 / c3 / c4, cold and warm, min / median / p95 over blocks.
  * cpu_baseline        : the CPU oracle as it stands, timed on this box's host cores on c2 (rank 0); also with one
                          thread, and on a sample of c5.

`--impl reference` times the oracle (the reference arm of this tier) on the same config and metric.
Nothing here reads /root/reference.  Only the cpu_baseline / reference legs touch `oracle/`.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "us_per_752x480_stereo_pair"
UNIT = "us/pair"
NOMINAL_HBM_GBS = 8000.0           # the data-sheet 8 TB/s (fraction reported against both peaks)
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback ("of fallback")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--blocks", type=int, default=50, help="back-to-back timed blocks of --steps steps; value = median block")
    ap.add_argument("--sets", type=int, default=64, help="distinct c2 input sets rotated through (cold inputs)")
    ap.add_argument("--no-batch64", action="store_true", help="skip the config-c5 (B=64 1080p) leg")
    ap.add_argument("--batch64-steps", type=int, default=30)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=0, help="0 = min(steps, 100)")
    ap.add_argument("--leg", default="all", choices=["all", "c2", "c5", "pre", "match"],
                    help="profiling aid: c5 = shortest possible c2 legs (13 c2 launches) then the batch-64 leg; "
                         "c2 = no batch-64 leg; pre = shortest c2 legs, then only the pre-processing kernel.  "
                         "The driver's bench line is --leg all.")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def kernels_sha():
    """Fingerprint of the device code the committed ncu table was captured from (first 12 hex digits of the sha256 of
    the kernel sources)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2607_01757_b200", "csrc")
    for f in ("dkd_kernels.cuh", "dkd_match.cu"):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:12]


def ncu_traffic(kernel, table="traffic_c5.csv"):
    """(dram read + write bytes of one launch of `kernel`, provenance) from the committed ncu --set full summary
    (profiles/traffic_*.csv: a text table copied from the capture, not something measured in this run).  The table
    records the fingerprint of the kernel sources it was captured from: `current` says whether it still matches."""
    tp = os.path.join(ROOT, "profiles", table)
    try:
        import csv
        for row in csv.DictReader(open(tp)):
            if row["kernel"] == kernel:
                sha = row.get("kernels_sha", "")
                return (int(row["dram_read_bytes"]) + int(row["dram_write_bytes"]),
                        {"file": "profiles/" + table, "kernels_sha": sha, "current": sha == kernels_sha()})
    except Exception:                                            # noqa: BLE001
        pass
    return None, None


class ClockSampler:
    """Samples SM clock + throttle reasons through NVML while `active` (DURING the timed regions)."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.active, self.stop = [], set(), False, False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        except Exception as e:                                   # noqa: BLE001
            self.nv = None
            self.err = str(e)

    def _run(self):
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self.stop:
            if self.active:
                try:
                    self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                    m = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                    for bit, n in names.items():
                        if m & bit:
                            self.reasons.add(n)
                except Exception:                                # noqa: BLE001
                    pass
                time.sleep(0.002)
            else:
                time.sleep(0.001)

    def __enter__(self):
        self.active = True
        return self

    def __exit__(self, *a):
        self.active = False

    def summary(self):
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": self.err}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def tensor_peak():
    """Dense fp16/bf16 tensor peak for a kernel timed alone: MEASURED_PEAKS.json bf16_tflops (burst), else the
    profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, burst; fp16 = bf16 rate)"
        except Exception:                                        # noqa: BLE001
            pass
    return 1590.0, "fallback (B200_PROFILING.md)"


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))


def credited_bytes(B, H, W, top_k, D, esz, kept, with_index=False):
    """Algorithmic bytes of one extract: score maps read once +
    4 sampled corner rows per kept keypoint + every output incl. padding."""
    score = B * H * W * 4
    corners = int(kept) * 4 * D * esz
    outputs = B * top_k * (8 + 4 + D * esz + (4 if with_index else 0)) + 4 * B
    return {"score": score, "corners": corners, "outputs": outputs, "total": score + corners + outputs}


def workload_name(cfg):
    return (f"{cfg.name}: B={cfg.B} {cfg.W}x{cfg.H} f32 score maps, r={cfg.r}, thresh={cfg.thresh}, top_k={cfg.top_k}, "
            f"T={cfg.T}; desc [{cfg.B},{cfg.Hd},{cfg.Wd},{cfg.D}] {cfg.desc_dtype} stride {cfg.stride}")


# ---------------------------------------------------------------------------------------------
def run_reference(args):
    """Reference arm of this tier = the CPU oracle as it stands, on the box's host cores (rank 0)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import numpy as np
    import oracle
    import synth
    cfg = synth.CONFIGS["c2"]
    nsets = 4
    sets = []
    for j in range(nsets):
        c = cfg.scaled(seed=cfg.seed + 1000 * j)
        score, desc = synth.make_inputs(c, device="cpu")
        sets.append((score.numpy(), desc.numpy()))

    def step(i):
        s, d = sets[i % nsets]
        return oracle.extract(s, d, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T)

    for i in range(max(args.warmup, 1)):
        step(i)
    t0 = time.perf_counter()
    for i in range(args.steps):
        step(i)
    dt = time.perf_counter() - t0
    ms = dt * 1e3 / args.steps
    val = ms * 1e3
    cores = oracle.num_threads()
    sample = "every step = the full c2 stereo pair (O1-O5 incl. descriptors); inputs in host memory"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": workload_name(cfg), "l2": "n/a (CPU)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import synth
    import paper_2607_01757_b200 as dkd
    from paper_2607_01757_b200.binding import OPT_PROFILE, OPT_USE_GRAPH

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — libdkd has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(x: float) -> float:
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    hbm_peak, peak_src = peaks()
    sampler = ClockSampler(local)
    cfg = synth.CONFIGS["c2"]
    esz = 2 if cfg.desc_dtype == "f16" else 4
    if args.leg in ("c5", "pre", "match"):
        args.sets, args.steps, args.warmup, args.e2e_steps, args.no_cpu_baseline = 1, 1, 3, 1, True
    if args.leg in ("pre", "match"):
        args.no_batch64 = True
    if args.leg == "c2":
        args.no_batch64 = True
    R = max(1, args.sets)
    K, Wm = args.steps, max(args.warmup, 3)

    # ---- c2: R distinct seeded input sets (cold inputs: touched bytes of R sets > L2) --------------
    ctx = dkd.DKD(cfg.B, cfg.H, cfg.W, cfg.top_k, cfg.D, device=local)
    stream = torch.cuda.current_stream(dev)
    calls, sets = [], []
    for j in range(R):
        c = cfg.scaled(seed=cfg.seed + 1000 * j + 100000 * rank)
        score, desc = synth.make_inputs(c, device=dev)
        sd = score.to(dev)
        out = ctx.alloc_outputs(cfg.B, cfg.top_k, desc, cfg.D, want_index=False, want_offsets=False)
        sets.append((sd, desc, out, score))
        calls.append(ctx.bind(sd, desc, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, out, stream))
    for f in calls:                                              # builds + caches one graph per set (untimed)
        f()
    torch.cuda.synchronize()
    kept = sum(int(s[2].count.sum()) for s in sets) / R
    cb = credited_bytes(cfg.B, cfg.H, cfg.W, cfg.top_k, cfg.D, esz, kept)

    def stats(xs):
        xs = sorted(xs)
        return {"min": xs[0], "median": xs[len(xs) // 2], "p95": xs[min(len(xs) - 1, int(len(xs) * 0.95))], "blocks": len(xs)}

    for i in range(Wm):
        calls[i % R]()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # The timed region is NB back-to-back blocks of exactly K steps each, an event between blocks, barrier + synchronize
    # on both sides of the series; `value` is the MEDIAN block (K = 20 is 0.35 ms of device time: a single block is
    # dominated by pipeline fill and box noise, the median of 50 is not), min and p95 are reported beside it.
    NB = args.blocks if args.leg not in ("c5", "pre", "match") else 1
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(NB + 1)]
    barrier()
    torch.cuda.synchronize()
    with sampler:
        t0 = time.perf_counter()
        evs[0].record(stream)
        it = 0
        for b in range(NB):
            for _ in range(K):
                calls[it % R]()
                it += 1
            evs[b + 1].record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
    barrier()
    block_ms = [evs[b].elapsed_time(evs[b + 1]) / K for b in range(NB)]
    bst = stats(block_ms)
    ms_step = max_over_ranks(bst["median"])
    wall_ms_step = max_over_ranks(wall * 1e3 / (K * NB))
    value_blocks = {"us_min": bst["min"] * 1e3 / world, "us_median": bst["median"] * 1e3 / world, "us_p95": bst["p95"] * 1e3 / world,
                    "blocks": NB, "steps_per_block": K, "us_mean_all_blocks": evs[0].elapsed_time(evs[NB]) * 1e3 / (K * NB) / world,
                    "what": "value = median over the blocks of (device time of K back-to-back steps) / K"}

    # single-shot latency (enqueue -> outputs complete), one pair at a time
    lat = []
    for i in range(min(200, max(K, 20)) if args.leg not in ("c5", "pre", "match") else 1):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        calls[i % R]()
        torch.cuda.synchronize()
        lat.append((time.perf_counter() - t0) * 1e6)
    lat.sort()

    # the paper's keypoint-cap sweep (caps 160 / 192 / 256 / 384, DKD runtime minimum at
    # 256 with its fixed 64-thread blocks): same c2 stereo pair, one graph launch per step, cap = top_k
    cap_sweep = None
    if args.leg == "all":
        cap_sweep = {}
        sd0, desc0 = sets[0][0], sets[0][1]
        for cap in (160, 192, 256, 384):
            outc = ctx.alloc_outputs(cfg.B, cap, desc0, cfg.D, want_index=False, want_offsets=False)
            fc = ctx.bind(sd0, desc0, cfg.stride, cfg.r, cfg.thresh, cap, cfg.T, outc, stream)
            for _ in range(20):
                fc()
            torch.cuda.synchronize()
            ev0.record(stream)
            for _ in range(500):
                fc()
            ev1.record(stream)
            torch.cuda.synchronize()
            cap_sweep[str(cap)] = ev0.elapsed_time(ev1) * 1e3 / 500
        cap_sweep["what"] = "us per 752x480 stereo pair vs keypoint cap (warm inputs: one input set)"

    # the other latency-bound configs (c1, c3, c4 = BASELINE.json configs[0], [2], [3]): us per call, one graph
    # launch per call, rotating through 16 seeded input sets each (the <= 50 us goal is reported
    # for them too)
    other_cfgs = None
    if args.leg == "all":
        other_cfgs = {}
        for name in ("c1", "c3", "c4"):
            cg = synth.CONFIGS[name]
            cx = dkd.DKD(cg.B, cg.H, cg.W, cg.top_k, cg.D, device=local)
            cl, keep = [], []
            for j in range(16):
                c = cg.scaled(seed=cg.seed + 1000 * j + 100000 * rank)
                sc, de = synth.make_inputs(c, device=dev)
                sdj = sc.to(dev)
                oj = cx.alloc_outputs(cg.B, cg.top_k, de, cg.D, want_index=False, want_offsets=False)
                keep.append((sdj, de, oj))
                cl.append(cx.bind(sdj, de, cg.stride, cg.r, cg.thresh, cg.top_k, cg.T, oj, stream))
            for f in cl:
                f()
            torch.cuda.synchronize()

            def blocks_us(fns, nb=20, per=48):
                es = [torch.cuda.Event(enable_timing=True) for _ in range(nb + 1)]
                for i in range(per):
                    fns[i % len(fns)]()
                es[0].record(stream)
                for b_ in range(nb):
                    for i in range(per):
                        fns[(b_ * per + i) % len(fns)]()
                    es[b_ + 1].record(stream)
                torch.cuda.synchronize()
                st_ = stats([es[b_].elapsed_time(es[b_ + 1]) * 1e3 / per for b_ in range(nb)])
                return {"min": st_["min"], "median": st_["median"], "p95": st_["p95"], "blocks": nb, "calls_per_block": per}

            cold = blocks_us(cl)
            warm = blocks_us(cl[:1])
            kept_c = sum(int(k[2].count.sum()) for k in keep) / 16
            other_cfgs[name] = {"us_per_call": cold["median"], "cold": cold, "warm": warm, "kept_keypoints": kept_c,
                                "workload": workload_name(cg),
                                "what": "us per call, one graph launch per call; cold = rotating through 16 seeded input sets, "
                                        "warm = one input set (L2-resident)"}
            del cl, keep
            cx.close()
        torch.cuda.empty_cache()

    # the same steps as plain stream launches (DKD_OPT_USE_GRAPH = 0: three PDL-linked launches per step)
    stream_us = stream_dev_us = graph_dev_us = None
    if args.leg not in ("c5", "pre", "match"):
        ctx.set_option(OPT_USE_GRAPH, 0)
        for i in range(Wm):
            calls[i % R]()
        barrier()
        torch.cuda.synchronize()
        ev0.record(stream)
        for i in range(K):
            calls[i % R]()
        ev1.record(stream)
        torch.cuda.synchronize()
        barrier()
        stream_us = max_over_ranks(ev0.elapsed_time(ev1) / K) * 1e3 / world
        # the device's own time per step: the same launches queued behind a sleeping kernel, so that the host's launch
        # rate (three launches per step from Python) does not limit them
        Kq = min(K, 1000)
        torch.cuda._sleep(int(30e-3 * 1.9e9))
        ev0.record(stream)
        for i in range(Kq):
            calls[i % R]()
        ev1.record(stream)
        torch.cuda.synchronize()
        barrier()
        stream_dev_us = max_over_ranks(ev0.elapsed_time(ev1) / Kq) * 1e3 / world
        ctx.set_option(OPT_USE_GRAPH, 1)
        torch.cuda._sleep(int(30e-3 * 1.9e9))
        ev0.record(stream)
        for i in range(Kq):
            calls[i % R]()
        ev1.record(stream)
        torch.cuda.synchronize()
        barrier()
        graph_dev_us = max_over_ranks(ev0.elapsed_time(ev1) / Kq) * 1e3 / world

    # the same steps with output buffers the cached graph has not seen: every call hands the library another output set,
    # so each launch goes through the kernel-node update path of the shape-keyed graph cache (no capture, no instantiate)
    fresh = None
    if args.leg not in ("c5", "pre", "match"):
        NF = 8
        fouts = [[ctx.alloc_outputs(cfg.B, cfg.top_k, sets[j][1], cfg.D, want_index=False, want_offsets=False) for _ in range(NF)]
                 for j in range(min(R, 8))]
        fcalls = [[ctx.bind(sets[j][0], sets[j][1], cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, o, stream) for o in fouts[j]]
                  for j in range(len(fouts))]
        st0 = ctx.graph_stats()
        for i in range(Wm):
            fcalls[i % len(fcalls)][i % NF]()
        barrier()
        torch.cuda.synchronize()
        ev0.record(stream)
        for i in range(K):
            fcalls[i % len(fcalls)][(i // len(fcalls)) % NF]()
        ev1.record(stream)
        torch.cuda.synchronize()
        barrier()
        st1 = ctx.graph_stats()
        fresh = {"value": max_over_ranks(ev0.elapsed_time(ev1) / K) * 1e3 / world, "unit": UNIT,
                 "graphs_instantiated_during": st1["instantiated"] - st0["instantiated"],
                 "node_updates_during": st1["updated"] - st0["updated"],
                 "what": "same steps, every call with another output set (pointer miss): the cached graph's kernel nodes are updated in place"}
        del fouts, fcalls

    # per-kernel device time at c2 (library measurement mode: plain launches + events)
    ctx.set_option(OPT_PROFILE, 1)
    kt2 = {}
    nprof = 50 if args.leg not in ("c5", "pre", "match") else 0
    for i in range(nprof + 5 if nprof else 0):
        calls[i % R]()
        d = ctx.profile_read()
        if i >= 5:
            for k, v in d.items():
                kt2[k] = kt2.get(k, 0.0) + v * 1e3 / nprof
    kt2_var = {}
    if nprof:                                                    # the same pair through the variants V1 / V2 (per-kernel times)
        sd_, desc_, out_, _ = sets[0]
        for name, kw in (("nms_iters2", dict(nms_iters=2)), ("score_bilinear", dict(score_mode=1))):
            acc = {}
            for i in range(25):
                ctx.extract(sd_, desc_, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, out=out_, want_index=False,
                            want_offsets=False, **kw)
                d = ctx.profile_read()
                if i >= 5:
                    for k, v in d.items():
                        acc[k] = acc.get(k, 0.0) + v * 1e3 / 20
            kt2_var[name] = acc
        calls[0]()                                               # restore set 0's outputs (the e2e leg compares against them)
        torch.cuda.synchronize()
    ctx.set_option(OPT_PROFILE, 0)

    # ---- e2e: HOST buffers through dkd_extract_host, copies inside the timed region -----------------
    Ke = args.e2e_steps or min(K, 100)
    host_sets = []
    for j in range(2):
        sd, desc, out, score = sets[j % R]
        host_sets.append((score.pin_memory(), desc.cpu().pin_memory(),
                          ctx.alloc_outputs(cfg.B, cfg.top_k, desc, cfg.D, want_index=False, want_offsets=False,
                                            device="cpu", pin=True)))
    # pinned descriptor map: dkd_extract_host samples the 4 corner rows of every kept keypoint in place
    # over PCIe instead of uploading the map (185 MB, of which 1.6 MB is ever read)
    h2d = cfg.B * cfg.H * cfg.W * 4 + cb["corners"]
    h2d_full = cfg.B * cfg.H * cfg.W * 4 + cfg.B * cfg.Hd * cfg.Wd * cfg.D * esz
    d2h = cfg.B * cfg.top_k * (8 + 4 + cfg.D * esz) + 4 * cfg.B

    def e2e_pass(resident, n):
        for i in range(3):
            s, d, o = host_sets[i % 2]
            ctx.extract_host(s, d, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, out=o, desc_resident=resident)
        barrier()
        torch.cuda.synchronize()
        blk = []
        for b_ in range(NBe):                                    # NBe blocks of n synchronised steps, host clock per block
            t0 = time.perf_counter()
            for i in range(n):
                s, d, o = host_sets[0 if resident else i % 2]
                ctx.extract_host(s, d, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T, out=o, desc_resident=resident)
            torch.cuda.synchronize()
            blk.append((time.perf_counter() - t0) * 1e6 / n)
        barrier()
        st_ = stats(blk)
        return max_over_ranks(st_["median"]), st_

    NBe = args.blocks if args.leg not in ("c5", "pre", "match") else 1
    with sampler:
        e2e_us, e2e_st = e2e_pass(False, Ke)
        e2e_res_us, e2e_res_st = e2e_pass(True, Ke)
    assert torch.equal(host_sets[0][2].count, sets[0][2].count.cpu())

    # ---- batch 64 (config c5): whole-path throughput + per-kernel roofline ---------------------------
    b64 = None
    roof = None
    if not args.no_batch64:
        c5 = synth.CONFIGS["c5"].scaled(seed=synth.CONFIGS["c5"].seed + 100000 * rank)
        need = c5.B * c5.Hd * c5.Wd * c5.D * 2 + 3 * c5.B * c5.H * c5.W * 4 + (3 << 30)
        del calls, host_sets
        sets.clear()
        ctx.close()
        torch.cuda.empty_cache()
        free, _ = torch.cuda.mem_get_info(dev)
        if free < need:
            b64 = {"skipped": f"needs {need >> 30} GiB of device memory, {free >> 30} GiB free"}
        else:
            ctx5 = dkd.DKD(c5.B, c5.H, c5.W, c5.top_k, c5.D, device=local)
            if os.environ.get("DKD_BENCH_NMS_UNIT"):             # tuning aid (not used by the driver's line)
                from paper_2607_01757_b200.binding import OPT_NMS_UNIT
                ctx5.set_option(OPT_NMS_UNIT, int(os.environ["DKD_BENCH_NMS_UNIT"]))
            if os.environ.get("DKD_BENCH_SEL_PREFETCH"):
                from paper_2607_01757_b200.binding import OPT_SEL_PREFETCH
                ctx5.set_option(OPT_SEL_PREFETCH, int(os.environ["DKD_BENCH_SEL_PREFETCH"]))
            score5 = synth.score_maps(c5.B, c5.H, c5.W, c5.seed, c5.base, c5.nblobs).to(dev)
            desc5 = synth.desc_maps(c5.B, c5.Hd, c5.Wd, c5.D, c5.seed, torch.float16, dev)
            out5 = ctx5.alloc_outputs(c5.B, c5.top_k, desc5, c5.D, want_index=False, want_offsets=False)
            call5 = ctx5.bind(score5, desc5, c5.stride, c5.r, c5.thresh, c5.top_k, c5.T, out5, stream)
            for _ in range(5):
                call5()
            torch.cuda.synchronize()
            K5 = max(args.batch64_steps, 3)
            barrier()
            torch.cuda.synchronize()
            with sampler:
                ev0.record(stream)
                for _ in range(K5):
                    call5()
                ev1.record(stream)
                torch.cuda.synchronize()
            barrier()
            ms5 = max_over_ranks(ev0.elapsed_time(ev1) / K5)
            kept5 = int(out5.count.sum())
            cb5 = credited_bytes(c5.B, c5.H, c5.W, c5.top_k, c5.D, 2, kept5)
            # per-kernel durations: measurement mode (plain launches, an event before/after each kernel)
            ctx5.set_option(OPT_PROFILE, 1)
            kt5 = {}
            with sampler:
                for i in range(K5 + 3):
                    call5()
                    d = ctx5.profile_read()
                    if i >= 3:
                        for k, v in d.items():
                            kt5[k] = kt5.get(k, 0.0) + v * 1e3 / K5
            ctx5.set_option(OPT_PROFILE, 0)
            gbs = cb5["total"] / (ms5 * 1e-3) / 1e9
            b64 = {
                "workload": workload_name(c5), "us_per_batch": ms5 * 1e3,
                "frames_per_s": sum_over_ranks(c5.B / (ms5 * 1e-3)), "keypoints_per_s": sum_over_ranks(kept5 / (ms5 * 1e-3)),
                "credited_bytes": cb5, "credited_gbs": gbs, "frac_of_hbm_peak": gbs / hbm_peak,
                "peak_gbs": hbm_peak, "peak_source": peak_src, "kernel_us": kt5, "steps": K5,
                "l2": "working set (0.53 GB of score maps + 34 GB descriptor map) exceeds L2",
            }
            # the dominant kernel and its algorithmic bytes:
            #   nms: the score maps, read once;  refine_gather: corner rows + outputs;  select: candidate keys
            algo = {"nms": cb5["score"], "refine_gather": cb5["corners"] + cb5["outputs"], "select": 0}
            dom = max(kt5, key=kt5.get)
            traffic, traffic_src = ncu_traffic(dom)
            ach = algo.get(dom, 0) / (kt5[dom] * 1e-6) / 1e9
            roof = {"bound": "hbm", "kernel": dom, "workload": "c5 (B=64 1920x1080)", "achieved": ach, "peak": hbm_peak,
                    "unit": "GB/s", "frac": ach / hbm_peak, "frac_nominal": ach / NOMINAL_HBM_GBS, "traffic": traffic,
                    "traffic_source": traffic_src, "peak_source": peak_src,
                    "algorithmic_bytes": algo.get(dom, 0), "kernel_us": kt5[dom],
                    "whole_path": {"achieved": gbs, "frac": gbs / hbm_peak, "frac_nominal": gbs / NOMINAL_HBM_GBS,
                                   "credited_bytes": cb5["total"]}}
            # the variants of SURVEY.md 8(f) f2 at c5: heat x reliability streamed as a second TMA stream (the NMS now
            # moves 8 B per pixel), and the validity mask (read only at candidates)
            var5 = None
            if args.leg in ("all", "c5") and world == 1:
                var5 = {}
                g5 = torch.Generator(device=dev).manual_seed(5)
                rel5 = torch.rand(score5.shape, generator=g5, device=dev) * 0.5 + 0.5
                msk5 = (torch.rand(score5.shape, generator=g5, device=dev) < 0.9).to(torch.uint8)
                ctx5.set_option(OPT_PROFILE, 1)
                for name, kw, bpp in (("reliability", dict(reliability=rel5), 8), ("mask", dict(valid_mask=msk5), 4),
                                      ("reliability+mask", dict(reliability=rel5, valid_mask=msk5), 8),
                                      ("nms_iters2", dict(nms_iters=2), 4),          # V1: suppress-and-recover NMS
                                      ("score_bilinear", dict(score_mode=1), 4)):   # V2: score at the refined point
                    acc = {}
                    for i in range(8):
                        ctx5.extract(score5, desc5, c5.stride, c5.r, 0.1 if "reliability" in name else c5.thresh, c5.top_k, c5.T,
                                     out=out5, want_index=False, want_offsets=False, **kw)
                        d = ctx5.profile_read()
                        if i >= 3:
                            for k, v in d.items():
                                acc[k] = acc.get(k, 0.0) + v * 1e3 / 5
                    nb = c5.B * c5.H * c5.W * bpp
                    var5[name] = {"kernel_us": acc, "nms_algorithmic_bytes": nb, "nms_gbs": nb / acc["nms"] / 1e3,
                                  "nms_frac_of_hbm_peak": nb / acc["nms"] / 1e3 / hbm_peak}
                ctx5.set_option(OPT_PROFILE, 0)
                del rel5, msk5
            b64["variants"] = var5
            del score5, desc5, out5, call5
            ctx5.close()
            torch.cuda.empty_cache()

    # ---- consumers of the descriptors: tcgen05 matching and the keyframe-database scan -----------
    match_leg, retr_leg = None, None
    if args.leg in ("all", "match") and world == 1:
        tf_peak, tf_src = tensor_peak()
        ctxm = dkd.DKD(2, 64, 128, 64, 0, device=local)

        def graph_time(fn, per_graph, reps):
            """GPU time of one call: `per_graph` calls captured into one graph (no Python between them), replayed."""
            fn(None)
            torch.cuda.synchronize()
            gph = torch.cuda.CUDAGraph()
            cs = torch.cuda.Stream(device=dev)
            with torch.cuda.stream(cs), torch.cuda.graph(gph, stream=cs):
                for _ in range(per_graph):
                    fn(cs)
            for _ in range(3):
                gph.replay()
            torch.cuda.synchronize()
            ev0.record(stream)
            for _ in range(reps):
                gph.replay()
            ev1.record(stream)
            torch.cuda.synchronize()
            return ev0.elapsed_time(ev1) * 1e3 / (reps * per_graph)

        match_leg = {"what": "dkd_match: P = 2 pairs (temporal + stereo, PAPER.md:132) of N x N x D fp16 descriptor sets, ratio 0.8; "
                             "us per call = k_match_tc + k_match_finalize, GPU time from graph replays",
                     "peak_tflops": tf_peak, "peak_source": tf_src, "sizes": {}}
        for (Nn, Dd) in ((256, 128), (1024, 128), (2048, 256), (4096, 128), (4096, 256)):
            A, Bm, cnta, cntb = synth.match_sets(2, Nn, Nn, Dd, seed=Nn + Dd)
            A, Bm, cnta, cntb = A.to(dev), Bm.to(dev), cnta.to(dev), cntb.to(dev)
            us = graph_time(lambda s_: ctxm.match(A, Bm, cnta, cntb, ratio=0.8, stream=s_), 10, 10)
            fl = 2.0 * Nn * Nn * Dd * 2
            match_leg["sizes"][f"N{Nn}_D{Dd}"] = {"us": us, "flops": fl, "tflops": fl / us / 1e6, "frac_of_tensor_peak": fl / us / 1e6 / tf_peak}
            if (Nn, Dd) in ((1024, 128), (4096, 256)):           # the mutual check: a second k_match_tc with the operands swapped
                usm = graph_time(lambda s_: ctxm.match(A, Bm, cnta, cntb, ratio=0.8, mutual=True, stream=s_), 10, 10)
                match_leg["sizes"][f"N{Nn}_D{Dd}"]["us_mutual"] = usm
                match_leg["sizes"][f"N{Nn}_D{Dd}"]["mutual_over_one_way"] = usm / us
        big = match_leg["sizes"]["N4096_D256"]
        match_leg["roofline"] = {"bound": "tensor", "kernel": "k_match_tc", "workload": "P=2 N=4096 D=256 fp16", "achieved": big["tflops"],
                                 "peak": tf_peak, "unit": "TFLOP/s", "frac": big["frac_of_tensor_peak"], "traffic": None,
                                 "peak_source": tf_src, "algorithmic_flops": big["flops"], "kernel_us": big["us"]}
        # f4: the elementwise consumers, per call (launch-bound: one small kernel each)
        nst = 1024
        gk = torch.Generator(device=dev).manual_seed(3)
        kl = torch.rand((nst, 2), generator=gk, device=dev) * 400 + 50
        kr = kl - torch.tensor([20.0, 0.0], device=dev)
        mt = torch.arange(nst, dtype=torch.int32, device=dev)
        cam = dict(fx=458.0, fy=457.0, cx=367.0, cy=248.0, baseline=0.11, d_min=1.0, z_min=0.3, z_max=30.0)
        Lf = torch.rand((nst, 3), generator=gk, device=dev) + 0.2
        covp = dict(scale=1.25, floor_px=0.0, fx=460.0, fy=455.0, lam=0.3, lam_min=0.05, sigma0=1.5 / 460.0)
        match_leg["stereo_validate_us"] = graph_time(lambda s_: ctxm.stereo_validate(kl, kr, mt, stream=s_, **cam), 20, 10)
        match_leg["cov_sqrt_info_us"] = graph_time(lambda s_: ctxm.cov_sqrt_info(Lf, stream=s_, **covp), 20, 10)
        match_leg["f4_what"] = "us per call on 1024 keypoints, GPU time from graph replays (20 calls per graph)"

        # the composed front-end of one stereo frame, device-resident: dkd_extract on B = 4 views
        # (L/R at t-1 and t) -> dkd_match P = 2 (temporal + stereo pair, ratio 0.8, mutual) on views of the extract outputs
        # -> dkd_stereo_validate; the whole chain captured in ONE caller graph and replayed
        frontend = {"what": "us per stereo frame: extract(B=4 752x480, 128-d f16) -> match(P=2, mutual) -> stereo_validate, one "
                            "caller graph, GPU time from graph replays; cap = keypoint cap (PAPER.md:171: 256)"}
        sq, dq = synth.stereo_sequence(cfg.H, cfg.W, cfg.D, seed=9, disparity=20, device=dev)
        sq = sq.to(dev)
        for cap in (256, 1024):
            cf_ = dkd.DKD(4, cfg.H, cfg.W, cap, cfg.D, device=local)
            of = cf_.alloc_outputs(4, cap, dq, cfg.D, want_index=False, want_offsets=False)

            def chain(s_, cf_=cf_, of=of, cap=cap):
                r_ = cf_.extract(sq, dq, 1, cfg.r, cfg.thresh, cap, cfg.T, out=of, stream=s_, want_index=False, want_offsets=False)
                m_, _ = cf_.match(r_.desc[0:2], r_.desc[1:3], r_.count[0:2], r_.count[1:3], ratio=0.8, mutual=True,
                                  want_sim=False, stream=s_)
                return cf_.stereo_validate(r_.kpts[1], r_.kpts[2], m_[1], stream=s_, max_reproj=1.5, **cam)

            us_f = graph_time(chain, 4, 25)
            v_ = chain(None)[0]
            torch.cuda.synchronize()
            frontend[f"cap{cap}"] = {"us": us_f, "keypoints": [int(x) for x in of.count.tolist()], "stereo_valid": int(v_.sum())}
            cf_.close()
        match_leg["frontend_frame_us"] = frontend
        del sq, dq
        # retrieval: AnyLoc-sized descriptors (32 x 384 = 12288); 20 000 keyframes = 492 MB > L2
        nk, Dg = 20000, 12288
        gq = torch.Generator(device=dev).manual_seed(11)
        db = torch.randn((nk, Dg), generator=gq, device=dev)
        db = (db / db.norm(dim=1, keepdim=True)).half()
        qv = db[17].float() * 0.8 + 0.6 * torch.nn.functional.normalize(torch.randn(Dg, generator=gq, device=dev), dim=0)
        qv = torch.nn.functional.normalize(qv, dim=0).half()
        us = graph_time(lambda s_: ctxm.retrieval_scan(db, qv, 50, 0.60, 16, stream=s_), 4, 10)
        _, cand, _, cnt = ctxm.retrieval_scan(db, qv, 50, 0.60, 16)
        torch.cuda.synchronize()
        assert int(cnt[0]) == 1 and int(cand[0]) == 17
        nbytes = nk * Dg * 2
        tr, tr_src = ncu_traffic("scan", "traffic_f3.csv")
        retr_leg = {"what": "dkd_retrieval_scan: one 12288-d fp16 query over 20000 keyframes (492 MB > L2), skip 50 newest, tau 0.60; "
                            "us per call = k_scan + k_select + k_cand_sims", "us": us,
                    "roofline": {"bound": "hbm", "kernel": "k_scan (+ select)", "workload": "n=20000 D=12288 fp16", "achieved": nbytes / us / 1e3,
                                 "peak": hbm_peak, "unit": "GB/s", "frac": nbytes / us / 1e3 / hbm_peak, "traffic": tr,
                                 "traffic_source": tr_src, "peak_source": peak_src, "algorithmic_bytes": nbytes, "kernel_us": us}}
        del db, qv
        ctxm.close()
        torch.cuda.empty_cache()

    # ---- fused input pre-processing kernel: stereo pair + batch 64 ----
    pre = None
    if args.leg in ("all", "pre"):
        pre = {}
        ctxp = dkd.DKD(2, 64, 64, 16, 0, device=local)
        for name, (Bp, Hq, Wq, dt, n_it) in {"stereo_752x480_mono_to_3ch_f32_grid32": (2, 480, 752, torch.float32, 200),
                                               "batch64_1920x1080_mono_to_3ch_f16_grid32": (64, 1080, 1920, torch.float16, 20)}.items():
            srcs = [torch.randint(0, 256, (Bp, Hq, Wq, 1), dtype=torch.uint8, device=dev) for _ in range(2 if Bp > 2 else 32)]
            Hp, Wp, _, _ = ctxp.padded_size(Hq, Wq, 32)
            outs = [torch.empty((Bp, 3, Hp, Wp), dtype=dt, device=dev) for _ in range(len(srcs))]
            kw = dict(mean=(0.485, 0.456, 0.406), inv_std=(4.367, 4.464, 4.444))
            for j in range(len(srcs)):
                ctxp.preprocess(srcs[j], 3, 32, out=outs[j], **kw)
            torch.cuda.synchronize()
            if Bp <= 2:                                          # launch-bound size: replay the launches from one
                gph = torch.cuda.CUDAGraph()                     # captured graph so that Python is not what is timed
                cs = torch.cuda.Stream(device=dev)
                with torch.cuda.stream(cs), torch.cuda.graph(gph, stream=cs):
                    for j in range(len(srcs)):
                        ctxp.preprocess(srcs[j], 3, 32, out=outs[j], stream=cs, **kw)
                gph.replay()
                torch.cuda.synchronize()
                reps = max(n_it // len(srcs), 1)
                ev0.record(stream)
                for _ in range(reps):
                    gph.replay()
                ev1.record(stream)
                torch.cuda.synchronize()
                us = ev0.elapsed_time(ev1) * 1e3 / (reps * len(srcs))
            else:
                ev0.record(stream)
                for i in range(n_it):
                    j = i % len(srcs)
                    ctxp.preprocess(srcs[j], 3, 32, out=outs[j], **kw)
                ev1.record(stream)
                torch.cuda.synchronize()
                us = ev0.elapsed_time(ev1) * 1e3 / n_it
            nbytes = Bp * Hq * Wq + Bp * 3 * Hp * Wp * outs[0].element_size()
            pre[name] = {"us": us, "algorithmic_bytes": nbytes, "gbs": nbytes / us / 1e3, "frac_of_hbm_peak": nbytes / us / 1e3 / hbm_peak,
                         "l2": f"rotates through {len(srcs)} buffer sets ({len(srcs) * nbytes / 1e6:.0f} MB)"}
            del srcs, outs
        ctxp.close()
        torch.cuda.empty_cache()

    # ---- CPU baseline: the oracle as it stands, on this box's host cores (rank 0, N = 1) -----------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle                                            # cpu_baseline leg only
        c = cfg.scaled(seed=cfg.seed)
        s_np, d_t = synth.make_inputs(c, device="cpu")
        s_np, d_np = s_np.numpy(), d_t.numpy()
        oracle.extract(s_np, d_np, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
        ts = []
        t_end = time.perf_counter() + 10.0
        while len(ts) < 200 and (time.perf_counter() < t_end or len(ts) < 3):
            t0 = time.perf_counter()
            oracle.extract(s_np, d_np, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
            ts.append(time.perf_counter() - t0)
        ts.sort()
        cpu = {"value": ts[len(ts) // 2] * 1e6, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"the full c2 stereo pair (O1-O5 incl. descriptors), median of {len(ts)} runs, host-resident inputs",
               "best": ts[0] * 1e6}
        # the same oracle on ONE thread, and on a sample of c5 (two figures, an oracle time beside c5)
        try:
            import ctypes
            gomp = ctypes.CDLL("libgomp.so.1")
            nthr = oracle.num_threads()
            gomp.omp_set_num_threads(1)
            t1 = []
            for _ in range(3):
                t0 = time.perf_counter()
                oracle.extract(s_np, d_np, cfg.stride, cfg.r, cfg.thresh, cfg.top_k, cfg.T)
                t1.append(time.perf_counter() - t0)
            gomp.omp_set_num_threads(nthr)
            cpu["one_thread"] = {"value": min(t1) * 1e6, "unit": UNIT, "cores": 1, "sample": "the full c2 stereo pair, best of 3"}
        except Exception as e:                                   # noqa: BLE001
            cpu["one_thread"] = {"error": str(e)}
        if not args.no_batch64:
            c5c = synth.CONFIGS["c5"]
            s5 = synth.score_maps(4, c5c.H, c5c.W, c5c.seed, c5c.base, c5c.nblobs).numpy()
            t0 = time.perf_counter()
            oracle.extract(s5, None, 1, c5c.r, c5c.thresh, c5c.top_k, c5c.T)
            dt5 = time.perf_counter() - t0
            cpu["c5"] = {"value": dt5 / 4 * c5c.B * 1e6, "unit": "us per batch of 64 (extrapolated)", "cores": oracle.num_threads(),
                         "sample": "steps O1-O3, O5 on 4 of the 64 frames of c5 (keypoints only: the 34 GB descriptor map is not "
                                   "materialised on the host), scaled to 64 frames"}

    if rank == 0:
        us_pair = ms_step * 1e3 / world
        line = {
            "metric": METRIC, "value": us_pair, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "l2": f"cold: steps rotate through {R} distinct seeded input sets "
                       f"({R * cb['total'] / 1e6:.0f} MB touched per rotation > 126 MB L2)",
                       "launch": "one cached CUDA-graph launch per step (3 kernels, programmatic dependent launch edges)", "parallelism": f"batch-sharded x{world}, no collective"},
            "frames_per_s": world * cfg.B / (ms_step * 1e-3), "keypoints_per_s": world * kept / (ms_step * 1e-3),
            "credited_bytes": cb, "credited_gbs": cb["total"] / (ms_step * 1e-3) / 1e9,
            "wall_ms_per_step": wall_ms_step, "value_blocks": value_blocks,
            "latency_us": {"median": lat[len(lat) // 2], "min": lat[0], "p95": lat[int(len(lat) * 0.95)],
                           "what": "single shot: enqueue -> stream idle, host clock"},
            "stream_launch": {"value": stream_us, "unit": UNIT, "queued_on_device": stream_dev_us, "graph_queued_on_device": graph_dev_us,
                              "what": "same steps with DKD_OPT_USE_GRAPH = 0: three PDL-linked launches per step instead of one graph launch "
                                      "(the NMS kernel of a step is launched under the previous step's refine/gather); queued_on_device = the "
                                      "same launches queued behind a sleeping kernel (the device's own time per step, no host launch-rate "
                                      "limit), graph_queued_on_device = the default graph launches measured the same way"},
            "fresh_buffers": fresh,
            "kernel_us_c2": kt2, "kernel_us_c2_variants": kt2_var,
            "clocks": sampler.summary(),
            "e2e": {"value": e2e_us / world, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": Ke, "blocks": e2e_st, "what": "median over blocks of `steps` calls; dkd_extract_host, pinned host buffers: score maps copied H2D, descriptor corner rows read "
                    "in place from the pinned map over PCIe (counted in h2d), every output stored by the kernels into the "
                    "pinned host tensors (counted in d2h); synchronised before return",
                    "descriptor_map_bytes_on_host": h2d_full - cfg.B * cfg.H * cfg.W * 4},
            "e2e_desc_resident": {"value": e2e_res_us / world, "unit": UNIT, "h2d_bytes_per_step": cfg.B * cfg.H * cfg.W * 4,
                                  "d2h_bytes_per_step": d2h,
                                  "what": "same, descriptor map left on the device by the previous call (network output)"},
            "gpu_launches": K * 3 * NB,
            "batch64": b64, "roofline": roof, "cpu_baseline": cpu, "match": match_leg, "retrieval": retr_leg, "preprocess": pre, "cap_sweep": cap_sweep, "other_configs": other_cfgs,
            "context": "paper: whole pipeline 29-47 FPS mono / 18-33 FPS stereo on Jetson AGX Orin (PAPER.md:5) — other hardware, whole system",
        }
        print(json.dumps(line), flush=True)
    sampler.stop = True
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
