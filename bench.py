#!/usr/bin/env python
"""bench.py -- events/s of the LST object-building chain on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W              # the CUDA path (this repo)
    python bench.py --impl reference --gpus N --steps K ...    # the CPU oracle, as it stands

Workload (config.workload): BASELINE.json config 5 at PU 200 -- batches of 16 independent
PU200-like events (config 3's generator, seeds 1000*PU + index, pLS seeds on), pipelined over CUDA
streams.  One STEP = one batch of 16 events through the whole chain (ingest/binning, MD, LS, T3,
T5, pT3, pT5, duplicate removal, track-candidate selection) = SURVEY.md section 8(a) rows a0..a6.

  value  : events/s with the batch inputs already resident in HBM (device pointers through the ABI)
  e2e    : events/s through the same C-ABI calls with HOST (pinned) buffers: H2D of the hits and
           seeds and D2H of the track candidates inside the timed region
  kernels / kernels_full_grid : per-kernel CUDA-event times (lst_ctx_kernel_times) of L2-flushed batches on one
           stream, in the configuration of the timed region (--blocks-per-sm, default 2: kernels of different
           batches share the SMs) and with every kernel filling the GPU (8 blocks per SM)
  roofline : the dominant kernel in the launch configuration of the timed region; roofline_full_grid: the same
           kernel filling the GPU on its own (8 blocks per SM)
  step_roofline : the whole timed step against the HBM and the issue-rate rooflines (BASELINE.json's metric)
  cpu_baseline : the oracle (oracle/) on the host cores over a bounded sample of the same events

Multi-GPU (N > 1): replicas only -- every rank runs its own batches (different seeds), no
collective on the data path; value = all ranks' events / max-over-ranks device time ("weak").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/sec at PU200-like occupancy (1 B200); fraction of HBM roofline"
UNIT = "events/s"
L2_BYTES = 126 << 20


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", choices=("b200", "reference"), default="b200")
    ap.add_argument("--pu", type=int, default=200)
    ap.add_argument("--workload", choices=("C5", "C6"), default="C5",
                    help="C5 = BASELINE.json configs[4] (the metric's workload); C6 = the strip-like second workload "
                         "of SURVEY.md 8(f)2 (lst_inputs.configs)")
    ap.add_argument("--truth-report", action="store_true",
                    help="run C4 and one batch of the workload through the CUDA path and print the synthetic-truth "
                         "metrics (PAPER.md:54-58, Figs. 3-4 in form) as JSON")
    ap.add_argument("--events", type=int, default=16, help="events per batch (= per step)")
    ap.add_argument("--streams", type=int, default=8, help="contexts / CUDA streams in flight")
    ap.add_argument("--blocks-per-sm", type=int, default=2,
                    help="lst_ctx_set_blocks_per_sm of every context: resident blocks per SM one kernel may take "
                         "(8 = every kernel fills the GPU; 1-2 let kernels of different batches share the SMs)")
    ap.add_argument("--batches", type=int, default=6, help="distinct input batches rotated through")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--stage-mask", type=lambda v: int(v, 0), default=None,
                    help="diagnostic: run the chain only up to a stage (CUTS.md section 9); written to config, "
                         "a line produced with it is not a benchmark of the whole path")
    ap.add_argument("--no-l2-flush", action="store_true",
                    help="diagnostic: per-kernel times with a warm L2; written to config")
    ap.add_argument("--profile-kernels-only", action="store_true",
                    help="run only the L2-flushed single-stream loop (the command ncu wraps)")
    return ap.parse_args()


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ---------------------------------------------------------------------------------------------
# inputs
# ---------------------------------------------------------------------------------------------
def make_batches(pu, n_events, n_batches, rank=0, world=1, config="C5"):
    """n_batches distinct batches of n_events C5 events (lst_inputs recipe); every rank
    takes its own event numbers (paper_2407_18231_b200.replicas: replicas only, no collective)."""
    from lst_inputs import make_config_event
    from lst_inputs.events import concat_events
    from paper_2407_18231_b200.replicas import event_indices

    out = []
    for idx in event_indices(rank, world, n_batches, n_events):
        evs = [make_config_event(config, pu=pu, index=i, seeds=True) for i in idx]
        out.append((evs, concat_events(evs)))
    return out


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed regions run."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self.stop_flag = threading.Event()
        self.active = threading.Event()
        self.err = None

    def run(self):
        try:
            import pynvml as nv

            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {
                nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
            }
            while not self.stop_flag.is_set():
                if self.active.is_set():
                    self.samples.append(int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                    for bit, name in names.items():
                        if r & bit:
                            self.reasons.add(name)
                time.sleep(0.002)
        except Exception as e:  # the clock record is evidence, not the product: report and go on
            self.err = repr(e)

    def summary(self):
        d = {"sm_mhz": int(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
             "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.err:
            d["error"] = self.err
        return d


# ---------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------
STAGE_OF_KERNEL = {"md": "md", "ls": "ls", "t3": "t3", "t5": "t5", "pt": "pt"}
# flops of the FIRST cut of a stage (every candidate evaluates at least that) and of the whole cut
# list (every accepted object evaluates all of it); counted from CUTS.md, no FMA.
FLOPS_FIRST = {"md": 19, "ls": 16, "t3": 28, "t5": 33, "pt3": 6, "pt5": 6}
FLOPS_FULL = {"md": 30, "ls": 64, "t3": 37, "t5": 44, "pt3": 100, "pt5": 107}


def algorithmic_work(name, s, n_sens):
    """(bytes, flops) one launch of kernel `name` must move / compute for batch summary `s`
    (compulsory traffic: every input array read once, every output written once)."""
    h, p = s["n_hits"], s["n_pls"]
    md, ls, t3, t5, p3, p5, tc = (s[k] for k in ("n_md", "n_ls", "n_t3", "n_t5", "n_pt3", "n_pt5", "n_tc"))
    idx = 5 * t5 + 5 * p5 + 3 * p3
    table = {
        # x, y, z + sensor id in, sorted (x, y, z, r) + (index, sensor) out, first hit of every sensor out;
        # seeds in, seed table out
        "ingest_count": 4 * h + 4 * h + 4 * 4 * n_sens + 32 * p + 56 * p,   # ids in, ranks out, 4 rows of counts out
        "ingest_scan": 2 * 4 * 4 * n_sens + 4 * n_sens,                      # counts in, slots and sens_begin out
        "scatter": 20 * h + 24 * h,                                          # ids, ranks, x, y, z in; sorted records out
        "md": 24 * h + 4 * n_sens + 20 * h,
        "md_place": 28 * h + 52 * md + 2 * n_sens,            # counts + stash in, MDs + module offsets out
        "ls": 28 * md + 8 * ls,
        "ls_place": 12 * md + 20 * ls + 16 * md,              # counts in, offsets + LSs out, index heads cleared
        "t3": 12 * ls + 16 * md + 44 * t3,
        "t5": 24 * t3 + 16 * md + 56 * t5 + 16 * md,          # + anchor bins and ranks
        "anchor_sort": 12 * md + 32 * md // 3,                # bins and ranks in, ~1/3 of the MDs are anchors
        "pt": 40 * p + 32 * md // 3 + 16 * (t3 + t5) + 8 * (p3 + p5),
        "pt_exact": 80 * (p3 + p5) + 12 * (p3 + p5),
        "pt_scan": 16 * p,
        "pt_place": 24 * (p3 + p5) + 4 * idx + 8 * idx,       # grouped by seed + the MD index of pT3, pT5, T5
        "rule1_pt5": 33 * p5,
        "rule2_pt3": 29 * p3,
        "rule3_t5": 25 * t5 + p,
        "tc_emit": 64 * tc + p5 + p3 + t5 + p,
    }
    st = STAGE_OF_KERNEL.get(name)
    flops = 0
    if st == "pt":  # one kernel builds pT3 and pT5
        for i, key, n_obj in ((4, "pt3", p3), (5, "pt5", p5)):
            flops += FLOPS_FIRST[key] * s["n_tests"][i] + (FLOPS_FULL[key] - FLOPS_FIRST[key]) * n_obj
    elif st:
        i = ("md", "ls", "t3", "t5").index(st)
        n_obj = (md, ls, t3, t5)[i]
        flops = FLOPS_FIRST[st] * s["n_tests"][i] + (FLOPS_FULL[st] - FLOPS_FIRST[st]) * n_obj
    return table.get(name, 0), flops


def workload_string(args):
    """config.workload: the same string from both arms (the driver compares them)."""
    if args.workload == "C6":
        return ("C6 PU%d: batches of %d strip-like events (SURVEY.md 8(f)2: C5's generator, 5 cm strips in the outer "
                "layers, r-z windows of lst_inputs.configs.C6_PARAMS), %d streams" % (args.pu, args.events, args.streams))
    return ("C5 PU%d: batches of %d PU200-like events (BASELINE.json configs[4]; generator of configs[2] with pLS "
            "seeds), %d streams" % (args.pu, args.events, args.streams))


def oracle_params(workload):
    import oracle

    if workload == "C6":
        from lst_inputs.configs import C6_PARAMS

        return oracle.default_params(**C6_PARAMS)
    return None


def workload_params(lst, workload, stage_mask=None):
    """Cut constants of the workload: CUTS.md defaults for C5; C6 opens the r-z windows to the strip length.
    stage_mask (--stage-mask, diagnostic only) cuts the chain short; it is recorded in the line's config."""
    kw = {}
    if workload == "C6":
        from lst_inputs.configs import C6_PARAMS

        kw.update(C6_PARAMS)
    if stage_mask is not None:
        kw["stage_mask"] = int(stage_mask)
    return lst.lst_default_params(**kw) if kw else None


def step_roofline(kernels, ms_step, hbm_gbs, peak_src, sm_max_mhz, args, E):
    """BASELINE.json's metric at step level: what the whole timed step reaches of the HBM roofline (sum of the kernels'
    algorithmic bytes / step time) and of the issue-rate roofline (sum of the executed warp instructions / step
    time).  Bytes are computed from this run's object counts; instruction counts need a profiler, so they come from the
    committed ncu capture (profiles/traffic.json) and only when it was taken on this workload."""
    alg = int(sum(k["alg_bytes"] for k in kernels))
    gbs = alg / (ms_step * 1e-3) / 1e9
    out = {"alg_bytes_per_step": alg, "gbs": round(gbs, 1), "hbm_peak_gbs": hbm_gbs, "hbm_frac": round(gbs / hbm_gbs, 4),
           "hbm_peak_source": peak_src + " copy bandwidth",
           "alg_bytes_source": "sum over the kernels of bench.algorithmic_work (every input read once, every output "
                               "written once) for this run's object counts",
           "ms_per_step": round(ms_step, 5), "warp_inst_per_step": None, "issue_frac": None, "dram_bytes_cold": None,
           "warp_inst_source": None}
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            cap = json.load(f)
        key = "kernels" if args.blocks_per_sm not in (0, 8) else "kernels_full_grid"
        names = [k["name"] for k in kernels]
        if cap.get("workload") == args.workload and cap.get("pu") == args.pu and cap.get("events") == E \
                and args.stage_mask is None and all(n in cap.get(key, {}) for n in names):
            wi = int(sum(cap[key][n].get("warp_inst", 0) for n in names))
            issue_peak = 148 * 4 * sm_max_mhz * 1e6  # 148 SMs x 4 schedulers x clock
            out["warp_inst_per_step"] = wi
            out["issue_frac"] = round(wi / (ms_step * 1e-3) / issue_peak, 4)
            out["dram_bytes_cold"] = int(sum(cap[key][n].get("dram_bytes", 0) for n in names))
            out["warp_inst_source"] = ("ncu capture %s (stored, not measured in this run; dram_bytes_cold = every kernel "
                                       "alone with caches flushed, an upper bound of the step's HBM traffic)"
                                       % cap.get("capture", "?"))
    return out


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def run_b200(args):
    import torch
    import torch.distributed as dist

    rank, world, local = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2407_18231_b200 import build as lst_build

    if rank == 0 or world == 1:
        lst_build.build()
    if world > 1:
        dist.barrier()
    import paper_2407_18231_b200 as lst
    from lst_inputs import make_config_geometry

    def barrier():
        if world > 1:
            dist.barrier()

    E, S, NB = args.events, max(1, args.streams), max(1, args.batches)
    geom, off, tgt = make_config_geometry(args.workload)
    n_sens = E * 2 * geom.n_modules
    t0 = time.time()
    batches = make_batches(args.pu, E, NB, rank, world, args.workload)
    gen_s = time.time() - t0

    g = lst.lst_load_geometry(geom.module_table(), off, tgt, workload_params(lst, args.workload, args.stage_mask))
    caps = lst.lst_default_caps(max_events=E)
    streams = [torch.cuda.Stream() for _ in range(S)]
    ctxs = [lst.lst_ctx_create(g, caps, st.cuda_stream) for st in streams]
    for c in ctxs:
        lst.lst_ctx_set_blocks_per_sm(c, args.blocks_per_sm)
    sampler = ClockSampler(local)
    sampler.start()

    # device-resident and pinned-host copies of every batch
    dev_in, host_in = [], []
    u16 = 2 * geom.n_modules <= 65536
    f_hit, f_pls = ("x", "y", "z", "sensor"), ("pt", "x0", "y0", "z0", "x1", "y1", "z1", "q")
    for _, b in batches:
        pin = {k: torch.from_numpy(np.ascontiguousarray(b[k])).pin_memory() for k in f_hit}
        pin_p = {k: torch.from_numpy(np.ascontiguousarray(b["pls"][k])).pin_memory() for k in f_pls}
        d = {k: v.cuda() for k, v in pin.items()}
        d_p = {k: v.cuda() for k, v in pin_p.items()}
        hd, keep_d = lst.make_hits(d["x"], d["y"], d["z"], d["sensor"], b["hit_offsets"])
        sd, keep_d = lst.make_pls(d_p, b["pls_offsets"], keep_d)
        # the host path sends the sensor ids as uint16 when they fit (lst_hits.sensor_u16): 14 bytes per hit over PCIe
        if u16:
            pin["sensor"] = torch.from_numpy(np.ascontiguousarray(b["sensor"].astype(np.uint16))).pin_memory()
        hh, keep_h = lst.make_hits(*(pin[k].numpy() for k in f_hit), b["hit_offsets"])
        sh, keep_h = lst.make_pls({k: v.numpy() for k, v in pin_p.items()}, b["pls_offsets"], keep_h)
        dev_in.append((hd, sd, keep_d, d, d_p))
        host_in.append((hh, sh, keep_h, pin, pin_p))
    in_bytes = [int(b["x"].shape[0]) * (14 if u16 else 16) + int(b["pls_offsets"][-1]) * 32 + 8 * (E + 1) + 64
                for _, b in batches]
    torch.cuda.synchronize()

    def pipelined(inputs, K, fetch):
        """K steps round-robin over the S contexts; returns (device ms, launches, last summaries)."""
        inflight = [False] * S
        launches = 0
        d2h = 0
        summ = [None] * S
        start = torch.cuda.Event(enable_timing=True)
        ends = [torch.cuda.Event(enable_timing=True) for _ in range(S)]
        start.record(streams[0])
        for st in streams:
            st.wait_event(start)

        def retire(c):
            nonlocal d2h
            summ[c] = lst.lst_ctx_sync(ctxs[c])  # status + counters of the batch this context ran
            if fetch:
                tc, _ = lst.lst_ctx_fetch_tc(ctxs[c], fetch[c], E)
                d2h += int(tc.shape[0]) * 64 + 4 * (4 * E + 1) + 160
            inflight[c] = False

        for i in range(K):
            c = i % S
            if inflight[c]:
                retire(c)
            h, s = inputs[i % NB][0], inputs[i % NB][1]
            lst.lst_ctx_run(ctxs[c], E, h, s)
            launches += lst.lst_ctx_launch_count(ctxs[c])
            inflight[c] = True
        for c in range(S):
            if inflight[c]:
                retire(c)
            ends[c].record(streams[c])
        torch.cuda.synchronize()
        return max(start.elapsed_time(e) for e in ends), launches, summ, d2h

    if not args.profile_kernels_only:
        # ---- value: inputs resident in HBM --------------------------------------------------
        pipelined(dev_in, max(args.warmup, S), None)
        torch.cuda.synchronize()
        barrier()
        sampler.active.set()
        ms, launches, summ, _ = pipelined(dev_in, args.steps, None)
        sampler.active.clear()
        barrier()
        # ---- e2e: host buffers, H2D + D2H inside ---------------------------------------------
        tc_pin = [torch.empty((caps.max_tc, 16), dtype=torch.int32).pin_memory().numpy() for _ in range(S)]
        pipelined(host_in, max(args.warmup, S), tc_pin)
        torch.cuda.synchronize()
        barrier()
        sampler.active.set()
        ms_e2e, _, _, d2h = pipelined(host_in, args.steps, tc_pin)
        sampler.active.clear()
        barrier()
        from paper_2407_18231_b200.replicas import max_over_ranks, sum_over_ranks

        ms, ms_e2e = max_over_ranks([ms, ms_e2e], device="cuda")  # the slowest rank sets the job's time
        launches = int(sum_over_ranks([launches], device="cuda")[0])

    # ---- per-kernel times: one stream, L2 flushed before every batch -----------------------------
    hbm_gbs, sm_max_mhz, peak_src = peaks()
    alu_peak_tflops = 148 * 128 * sm_max_mhz * 1e6 / 1e12  # FP32 lanes x clock, no FMA (CUTS.md section 0)
    flush = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device="cuda")
    reps = 3 if args.profile_kernels_only else 12

    def per_kernel_pass(blocks_per_sm):
        """Single-stream loop with CUDA events between the kernels (no graph), L2 flushed before every batch."""
        lst.lst_ctx_set_blocks_per_sm(ctxs[0], blocks_per_sm)
        lst.lst_ctx_set_timing(ctxs[0], True)
        per_kernel = {}
        order = []
        ksum = None
        for r in range(reps + 2):
            b = r % NB
            with torch.cuda.stream(streams[0]):
                if not args.no_l2_flush:
                    flush.zero_()
            lst.lst_ctx_run(ctxs[0], E, dev_in[b][0], dev_in[b][1])
            s_b = lst.lst_ctx_sync(ctxs[0])
            if r < 2:
                continue  # warm-up
            for name, t in lst.lst_ctx_kernel_times(ctxs[0]):
                if name not in per_kernel:
                    per_kernel[name] = []
                    order.append(name)
                w = algorithmic_work(name, s_b, n_sens)
                per_kernel[name].append((t, w[0], w[1]))
            ksum = s_b
        lst.lst_ctx_set_timing(ctxs[0], False)
        kernels = []
        tot_ms = sum(float(np.mean([v[0] for v in per_kernel[n]])) for n in order)
        for n in order:
            t = float(np.mean([v[0] for v in per_kernel[n]]))
            by = float(np.mean([v[1] for v in per_kernel[n]]))
            fl = float(np.mean([v[2] for v in per_kernel[n]]))
            gbs = by / (t * 1e-3) / 1e9 if t > 0 else 0.0
            tf = fl / (t * 1e-3) / 1e12 if t > 0 else 0.0
            kernels.append({"name": n, "ms": round(t, 5), "share": round(t / tot_ms, 4), "alg_bytes": int(by),
                            "gbs": round(gbs, 1), "hbm_frac": round(gbs / hbm_gbs, 4), "alg_flops": int(fl),
                            "tflops": round(tf, 3), "alu_frac": round(tf / alu_peak_tflops, 4)})
        return kernels, ksum

    sampler.active.set()
    kernels, ksum = per_kernel_pass(args.blocks_per_sm)  # the launch configuration of the timed region
    kernels_alone = None
    if not args.profile_kernels_only and args.blocks_per_sm not in (0, 8):
        kernels_alone, _ = per_kernel_pass(8)            # every kernel filling the GPU on its own
        lst.lst_ctx_set_blocks_per_sm(ctxs[0], args.blocks_per_sm)
    sampler.active.clear()
    # DRAM traffic and executed warp instructions of the dominant kernel cannot be measured without a profiler:
    # they come from the committed ncu --set full capture (profiles/traffic.json), and only when that capture was
    # taken on this workload; the field says so
    def make_roof(kernels, cap_key="kernels"):
        top = max(kernels, key=lambda k: k["ms"])
        if top["alu_frac"] >= top["hbm_frac"]:
            roof = {"bound": "alu", "kernel": top["name"], "achieved": top["tflops"], "peak": round(alu_peak_tflops, 2),
                    "unit": "TFLOP/s", "frac": top["alu_frac"], "traffic": None,
                    "peak_source": "148 SM x 128 FP32 lanes x %.0f MHz, 1 flop/lane/clk (no FMA)" % sm_max_mhz}
        else:
            roof = {"bound": "hbm", "kernel": top["name"], "achieved": top["gbs"], "peak": hbm_gbs, "unit": "GB/s",
                    "frac": top["hbm_frac"], "traffic": None, "peak_source": peak_src + " copy bandwidth"}
        roof["ms"] = top["ms"]
        traffic_path = os.path.join(ROOT, "profiles", "traffic.json")
        roof["traffic_source"] = None
        if os.path.exists(traffic_path):
            with open(traffic_path) as f:
                cap = json.load(f)
            if cap.get("workload") == args.workload and cap.get("pu") == args.pu and cap.get("events") == E \
                    and top["name"] in cap.get(cap_key, {}):
                k = cap[cap_key][top["name"]]
                roof["traffic"] = k.get("dram_bytes")
                roof["traffic_source"] = "ncu capture %s (stored, not measured in this run)" % cap.get("capture", "?")
                if k.get("warp_inst"):  # issue-rate roofline: 148 SMs x 4 schedulers x clock
                    issue_peak = 148 * 4 * sm_max_mhz * 1e6
                    roof["issue_frac"] = round(k["warp_inst"] / (top["ms"] * 1e-3) / issue_peak, 4)
                    roof["warp_inst"] = k["warp_inst"]
        return roof

    # `roofline`: the dominant kernel in the LAUNCH CONFIGURATION OF THE TIMED REGION (--blocks-per-sm), timed alone on
    # one stream.  With 1..4 blocks per SM a kernel takes only that share of every SM by design and leaves the rest to
    # the kernels of other batches, so this is the kernel as the step runs it, not the most the kernel can reach:
    # `roofline_full_grid` is the same kernel filling the GPU on its own (8 blocks per SM).
    cfg = "%d blocks per SM per kernel, kernel alone on one stream, L2 " + ("warm" if args.no_l2_flush else "flushed")
    roof = make_roof(kernels, "kernels" if args.blocks_per_sm not in (0, 8) else "kernels_full_grid")
    roof["launch"] = cfg % (args.blocks_per_sm or 8) + " (the configuration of the timed region)"
    roof_full = None
    if kernels_alone:
        roof_full = make_roof(kernels_alone, "kernels_full_grid")
        roof_full["launch"] = cfg % 8
    sampler.stop_flag.set()
    sampler.join(timeout=2)

    if args.profile_kernels_only:
        if rank == 0:
            print(json.dumps({"kernels": kernels, "summary": ksum}))
        for c in ctxs:
            lst.lst_free(c)
        lst.lst_free(g)
        return

    # ---- PCIe: what a pinned host -> device copy of one step's input reaches on this box, next to what e2e moved ----
    nbytes = int(np.mean(in_bytes))
    src = [torch.zeros(nbytes, dtype=torch.uint8).pin_memory() for _ in range(S)]
    dst = [torch.empty(nbytes, dtype=torch.uint8, device="cuda") for _ in range(S)]

    def h2d_rate(n_streams, reps):
        """GB/s of `reps` pinned host -> device copies of one step's input per stream, n_streams streams at once."""
        t0 = torch.cuda.Event(enable_timing=True)
        t1 = [torch.cuda.Event(enable_timing=True) for _ in range(n_streams)]
        torch.cuda.synchronize()
        t0.record(streams[0])
        for k in range(n_streams):
            streams[k].wait_event(t0)
            with torch.cuda.stream(streams[k]):
                for r in range(reps):
                    dst[k].copy_(src[k], non_blocking=True)
            t1[k].record(streams[k])
        torch.cuda.synchronize()
        return n_streams * reps * nbytes / (max(t0.elapsed_time(e) for e in t1) * 1e-3) / 1e9

    h2d_rate(S, 2)
    h2d_one, h2d_peak = h2d_rate(1, 20), h2d_rate(S, 10)
    e2e_gbs = (nbytes + d2h / args.steps) / (ms_e2e / args.steps * 1e-3) / 1e9
    pcie = {"pcie_h2d_peak_gbs": round(h2d_peak, 1), "pcie_h2d_one_stream_gbs": round(h2d_one, 1),
            "pcie_gbs": round(e2e_gbs, 1), "pcie_frac": round(e2e_gbs / max(h2d_peak, h2d_one), 3),
            "pcie_note": "peak = pinned cudaMemcpyAsync host -> device of one step's input size, 10 copies on each of "
                         "the %d streams at once (one stream alone: 20 copies), measured in this run; pcie_gbs = (H2D + "
                         "D2H bytes per step) / e2e ms per step; pcie_frac = pcie_gbs / the larger of the two" % S}

    # ---- CPU baseline (rank 0, N = 1 only) -------------------------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_rate(batches[0][0][:E], geom, off, tgt, params=oracle_params(args.workload))

    n_hits = [int(b["x"].shape[0]) for _, b in batches]
    line = {
        "metric": METRIC, "value": round(world * args.steps * E / (ms * 1e-3), 1), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "warmup_effective": max(args.warmup, S),
        "ms_per_step": round(ms / args.steps, 5),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {
            "workload": workload_string(args),
            "events_per_step": E, "hits_per_event": int(np.mean(n_hits) / E), "pls_per_event": ksum["n_pls"] // E,
            "modules": int(geom.n_modules), "parallelism": "replicas x%d, no collective" % world,
            "streams": S, "blocks_per_sm": args.blocks_per_sm,
            "l2": "inputs rotate over %d distinct batches + %d context workspaces (> 126 MB L2); per-kernel "
                  "times taken with an L2 flush (252 MB write) before every batch" % (NB, S),
            "objects_per_step": {k: ksum["n_" + k] for k in ("md", "ls", "t3", "t5", "pt3", "pt5", "tc")},
            "tests_per_step": dict(zip(("md", "ls", "t3", "t5", "pt3", "pt5"), ksum["n_tests"])),
            "near_threshold_per_step": dict(zip(("md", "ls", "t3", "t5", "pt3", "pt5"), ksum["near"])),
            # north_star states the 0.01 % bar against objects; reading N2 checks it against candidates
            "near_frac_of_candidates": {k: (round(n / t, 9) if t else None) for k, n, t in
                                        zip(("md", "ls", "t3", "t5", "pt3", "pt5"), ksum["near"], ksum["n_tests"])},
            "near_frac_of_objects": {k: (round(n / ksum["n_" + k], 9) if ksum["n_" + k] else None) for k, n in
                                     zip(("md", "ls", "t3", "t5", "pt3", "pt5"), ksum["near"])},
            "generation_s": round(gen_s, 1),
            "stage_mask": hex(args.stage_mask) if args.stage_mask is not None else "default (0x3f, whole chain)",
            "l2_flush_per_kernel_pass": not args.no_l2_flush,
        },
        "e2e": {"value": round(world * args.steps * E / (ms_e2e * 1e-3), 1), "unit": UNIT,
                "h2d_bytes_per_step": int(np.mean(in_bytes)), "d2h_bytes_per_step": int(d2h / args.steps),
                "input_format": "x, y, z float32 + sensor %s per hit; 8 x 4 bytes per seed" % ("uint16" if u16 else "int32"),
                "ms_per_step": round(ms_e2e / args.steps, 5), **pcie},
        "gpu_launches": launches,
        "clocks": sampler.summary(),
        "roofline": roof,
        "step_roofline": step_roofline(kernels, ms / args.steps, hbm_gbs, peak_src, sm_max_mhz, args, E),
        "kernels": kernels,
        "roofline_full_grid": roof_full,
        "kernels_full_grid": kernels_alone,
        "objects_per_s": {k: round(ksum["n_" + k] / (ms / args.steps * 1e-3), 1)
                          for k in ("md", "ls", "t3", "t5", "pt3", "pt5", "tc")},
        "cpu_baseline": cpu,
    }
    if rank == 0:
        print(json.dumps(line))
    for c in ctxs:
        lst.lst_free(c)
    lst.lst_free(g)
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------
# the CPU oracle: cpu_baseline leg and --impl reference
# ---------------------------------------------------------------------------------------------
def oracle_rate(events, geom, off, tgt, single=True, params=None):
    """Times oracle.run_event (as it stands, one thread per event) over `events` on the host cores."""
    from concurrent.futures import ThreadPoolExecutor

    import oracle

    oracle.build()
    cores = os.cpu_count() or 1
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        pass
    threads = max(1, min(cores, len(events)))

    def one(ev):
        r = oracle.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, params)
        return len(r["tc"])

    t_single = float("nan")
    if single:
        t0 = time.perf_counter()
        one(events[0])
        t_single = time.perf_counter() - t0
    t0 = time.perf_counter()
    with ThreadPoolExecutor(threads) as ex:  # ctypes releases the GIL inside the C call
        list(ex.map(one, events))
    wall = time.perf_counter() - t0
    return {"value": round(len(events) / wall, 3), "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": "%d events of the first batch, one oracle.run_event per event, %d threads (host has %d "
                      "cores); single thread: %.3f events/s" % (len(events), threads, cores, 1.0 / t_single),
            "single_thread_value": round(1.0 / t_single, 3)}


def run_reference(args):
    """The oracle as it stands on the host cores: same config, metric and unit as the CUDA arm.
    Each step is a bounded sample of the workload: `cores` events of the step's batch."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    from lst_inputs import make_config_geometry

    geom, off, tgt = make_config_geometry(args.workload)
    cores = os.cpu_count() or 1
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        pass
    per_step = max(1, min(cores, args.events))
    oparams = oracle_params(args.workload)
    # keep the whole run within a few minutes: ~1.5 s of one core per PU200 event
    steps = max(1, min(args.steps, 20))
    warm = max(0, min(args.warmup, 1))
    batches = make_batches(args.pu, per_step, 2, config=args.workload)
    for _ in range(warm):
        oracle_rate(batches[0][0], geom, off, tgt, single=False, params=oparams)
    t0 = time.perf_counter()
    res = None
    for i in range(steps):
        res = oracle_rate(batches[i % 2][0], geom, off, tgt, single=False, params=oparams)
    wall = time.perf_counter() - t0
    n_ev = steps * per_step
    value = round(n_ev / wall, 3)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": args.warmup, "warmup_effective": warm, "steps_requested": args.steps,
        "ms_per_step": round(wall / steps * 1e3, 3), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_string(args), "events_per_step": per_step,
                   "note": "each step is a bounded sample of %d events of the step's batch" % per_step},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": res["cores"], "kind": "oracle",
                         "sample": "%d steps x %d events, oracle.run_event, %d threads" % (steps, per_step,
                                                                                           res["cores"])},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_truth_report(args):
    """synthetic-truth metrics of the track candidates the CUDA path returns (PAPER.md:54-58,
    Figs. 3-4 in form, not in values): C4 (prompt + displaced tracks) and one batch of the workload."""
    import torch

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    from paper_2407_18231_b200 import build as lst_build

    lst_build.build()
    import paper_2407_18231_b200 as lst
    from lst_inputs import make_config_event, make_config_geometry
    from lst_inputs.events import concat_events
    from lst_inputs.truth_metrics import merge_metrics, track_candidate_metrics

    out = {}
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    g = lst.lst_load_geometry(geom.module_table(), off, tgt)
    res = lst.lst_run_event(g, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    lst.lst_free(g)
    out["C4"] = {"all": track_candidate_metrics(res, ev), "with_outer_tracker_hits": track_candidate_metrics(res, ev, classes=(0, 1, 2)),
                 "T5_only": track_candidate_metrics(res, ev, classes=(2,))}
    geom, off, tgt = make_config_geometry(args.workload)
    evs = [make_config_event(args.workload, pu=args.pu, index=i, seeds=True) for i in range(args.events)]
    b = concat_events(evs)
    g = lst.lst_load_geometry(geom.module_table(), off, tgt, workload_params(lst, args.workload))
    ctx = lst.lst_ctx_create(g, lst.lst_default_caps(max_events=args.events), torch.cuda.Stream().cuda_stream)
    h, keep = lst.make_hits(b["x"], b["y"], b["z"], b["sensor"], b["hit_offsets"])
    s, keep = lst.make_pls(b["pls"], b["pls_offsets"], keep)
    lst.lst_ctx_run(ctx, len(evs), h, s)
    lst.lst_ctx_sync(ctx)
    per_ev = [lst.lst_ctx_fetch_event(ctx, i) for i in range(len(evs))]
    lst.lst_free(ctx)
    lst.lst_free(g)
    key = "%s_PU%d_x%d" % (args.workload, args.pu, len(evs))
    out[key] = {"all": merge_metrics([track_candidate_metrics(r, e) for r, e in zip(per_ev, evs)]),
                "with_outer_tracker_hits": merge_metrics([track_candidate_metrics(r, e, classes=(0, 1, 2))
                                                          for r, e in zip(per_ev, evs)])}
    print(json.dumps({"truth_report": out, "source": "track candidates fetched through the C ABI (CUDA path)"}))


def main():
    args = parse_args()
    if args.truth_report:
        run_truth_report(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
