#!/usr/bin/env python
"""bench.py -- throughput of the ODB hot path (group -> align -> collate) on B200.

One "step" = one pass of the whole hot path (window fill, segmented
sort, greedy successor, list ranking, cross-rank reduction, split/overflow, step totals, offsets,
collation with valid-token counts) through ``odb_run`` over one batch of synthetic input that is
already resident in HBM.  Default workload = BASELINE.json configs[4] (the throughput sweep, the
largest config, on which north_star states its target), cell CV=1.0 / budget=65536, paper rule
(THRESHOLD), join mode.  The default run also times the nine (CV, budget) cells of configs[4] and configs[1..3] (key
``sweep``; ``--no-sweep`` skips it, ``--sweep`` adds the MAXFIT_ASC rule) and the paper's operating point, a
1024-sample grouping buffer per rank (key ``paper_operating_point``); ``--config k`` picks another
BASELINE.json config, ``--buffer-size`` another window.

Prints ONE JSON line (rank 0).  Extra objects: ``roofline`` (collate kernel, CUDA events on the
launching stream inside the timed region), ``e2e`` (odb_run_host with pinned HOST buffers, copies
inside the timed region), ``cpu_baseline`` (the oracle, as it stands, on a bounded sample on the
box's host cores), ``clocks`` (nvidia-smi sampled during the timed region).

``--impl reference`` times the CPU oracle instead (rank 0 only), per the tier contract.
Multi-GPU: the path does not shard across GPUs (north_star: virtual ranks on ONE GPU, no inter-GPU
collectives) -> "replicas only": N independent replicas, max-over-ranks time, value = N x units / t.
``--gpus N`` without a torchrun environment starts the N processes itself (one per GPU, NCCL rendezvous on
127.0.0.1) and fails loudly when the box has fewer than N devices; under torchrun WORLD_SIZE must equal N.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import odb_inputs as I  # noqa: E402

METRIC = "samples/s grouped+aligned+collated (with tokens/s and achieved HBM GB/s vs peak)"
UNIT = "samples/s"
RULE_NAMES = {0: "threshold", 1: "maxfit_asc"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (0-based)")
    ap.add_argument("--cv", type=float, default=1.0)
    ap.add_argument("--budget", type=int, default=None)
    ap.add_argument("--rule", type=int, default=0)
    ap.add_argument("--join", type=int, default=1)
    ap.add_argument("--buffer-size", type=int, default=None, help="per-round window per rank (0 = whole stream)")
    ap.add_argument("--sweep", action="store_true", help="the sweep also runs the MAXFIT_ASC rule on every cell")
    ap.add_argument("--no-sweep", action="store_true", help="skip the sweep cells and the paper operating point")
    ap.add_argument("--shard-ranks", action="store_true",
                    help="SURVEY.md 8(f) F1: split the job's virtual ranks over the N GPUs (strong scaling; per-round "
                         "all_gather + all_reduce over NCCL) instead of N independent replicas")
    ap.add_argument("--per-round-exchange", action="store_true",
                    help="--shard-ranks: one exchange per protocol round (P:52) instead of the batched exchange")
    ap.add_argument("--pipeline", type=int, default=0,
                    help="measure N contexts driven round-robin on N streams (planning of one step beside the collate "
                         "kernel of another); extra key 'pipelined'")
    ap.add_argument("--host-staging-elems", type=int, default=None,
                    help="arena elements per device staging piece of odb_run_host (ODB_OPT_HOST_STAGING_ELEMS)")
    ap.add_argument("--collate-bulk", action="store_true",
                    help="time the bulk-store (cp.async.bulk) form of the collate kernel instead of the adopted one")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample-ranks", type=int, default=16)
    ap.add_argument("--ref-sample-ranks", type=int, default=2)
    return ap.parse_args()


def workload_name(args, wl):
    b = wl.params["budget"]
    if args.config == 4:
        return ("configs[4] throughput sweep cell: %d virtual ranks x %d samples, lognormal(mean 2048, CV %g), budget %d"
                % (wl.n_ranks, wl.n_samples // max(wl.n_ranks, 1), args.cv, b))
    return "configs[%d] %s: %d virtual ranks, %d samples, budget %d" % (args.config, wl.name, wl.n_ranks,
                                                                         wl.n_samples, b)


def make_wl(args, **over):
    kw = dict(rule=args.rule, join_mode=args.join, budget=args.budget)
    if args.config == 4:
        kw["cv"] = args.cv
    kw.update(over)
    wl = I.make_workload(args.config, **kw)
    if args.buffer_size is not None:
        wl.params["buffer_size"] = args.buffer_size
    return wl


def algorithmic_bytes(real_tokens, padded_elems):
    """4 B read per real token + 13 B written per padded element (3 x int32 + uint8)."""
    return 4 * int(real_tokens) + 13 * int(padded_elems)


# --------------------------------------------------------------------------------------------
# clocks sampling (B200_PROFILING.md "clocks DURING the timed region")
# --------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
        time.sleep(0.25)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
                pw.append(float(f[3]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs: torch copy, read+write bytes)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(workload_key):
    """dram bytes per collate launch from the committed ncu --set full summary (profiles/), keyed by cell, or
    None: a cell that has no capture of the committed kernel reports null, never another cell's constant."""
    p = os.path.join(ROOT, "profiles", "collate_traffic.txt")
    try:
        with open(p) as f:
            for line in f:
                if line.startswith("#") or ":" not in line:
                    continue
                k, v = line.split(":", 1)
                if k.strip() == workload_key:
                    return float(v.split()[0])
    except OSError:
        pass
    return None


# --------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline and --impl reference).  The only place bench.py touches oracle/.
# --------------------------------------------------------------------------------------------
def oracle_time_once(wl, tokens):
    """One pass of the oracle (plan + collation of every slot) over `wl`; returns seconds."""
    from oracle import odb_oracle as O
    p = wl.params
    t0 = time.perf_counter()
    plan = O.OraclePlan(wl.lengths, wl.rank_ptr, **p)
    plan.collate_all(tokens, wl.sample_ptr[:-1], wl.span_ptr, wl.span_lo, wl.span_hi, pad_id=p["pad_id"],
                     ignore_index=p["ignore_index"], shift_labels=p["shift_labels"])
    dt = time.perf_counter() - t0
    return dt, plan


def cpu_baseline(args, n_ranks_sample):
    from oracle import odb_oracle as O
    O.build()
    full = I.bj_config(args.config)
    R = min(n_ranks_sample, full["R"])
    wl = make_wl(args, n_ranks=R)
    tokens = wl.tokens()          # host-side hash, untimed (token generation is excluded on both sides)
    dt, plan = oracle_time_once(wl, tokens)
    return {"value": plan.samples_emitted / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%d of %d virtual ranks of the same recipe (%d samples, %d real tokens), one pass, %.2f s; "
                      "single thread of %d host cores" % (R, full["R"], plan.samples_emitted, plan.real_tokens, dt,
                                                          os.cpu_count() or 0),
            "tokens_per_s": plan.real_tokens / dt, "seconds": dt}, wl


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import odb_oracle as O
    O.build()
    full = I.bj_config(args.config)
    R = min(args.ref_sample_ranks, full["R"])
    wl = make_wl(args, n_ranks=R)
    tokens = wl.tokens()
    for _ in range(args.warmup):
        oracle_time_once(wl, tokens)
    tot, plan = 0.0, None
    for _ in range(args.steps):
        dt, plan = oracle_time_once(wl, tokens)
        tot += dt
    ms = 1e3 * tot / max(args.steps, 1)
    val = plan.samples_emitted / (ms / 1e3)
    sample = "each step = %d of %d virtual ranks of the same recipe (%d samples, %d real tokens)" % (
        R, full["R"], plan.samples_emitted, plan.real_tokens)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": workload_name(args, make_wl_desc(args)), "rule": RULE_NAMES[args.rule],
                       "join_mode": args.join, "sample": sample},
            "tokens_per_s": plan.real_tokens / (ms / 1e3),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class _Desc:
    pass


def make_wl_desc(args):
    """Cheap stand-in with the full config's shape for workload_name (no arrays drawn)."""
    c = I.bj_config(args.config)
    d = _Desc()
    d.n_ranks, d.n_samples, d.name = c["R"], c["R"] * c["n"], c["name"]
    d.params = {"budget": args.budget if args.budget is not None else c["budget"]}
    return d


# --------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------
class DeviceInputs:
    def __init__(self, wl, device, P):
        import torch
        t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dt).to(device)
        self.lengths = t(wl.lengths, torch.int32)
        self.sample_ptr = t(wl.sample_ptr, torch.int64)
        self.span_ptr = t(wl.span_ptr, torch.int64)
        z = torch.zeros(1, dtype=torch.int32, device=device)
        self.span_lo = t(wl.span_lo, torch.int32) if len(wl.span_lo) else z
        self.span_hi = t(wl.span_hi, torch.int32) if len(wl.span_hi) else z
        self.tokens = torch.empty(wl.n_tokens + 16, dtype=torch.int32, device=device)
        P.odb_synth_tokens(self.tokens, 0, wl.n_tokens, wl.token_seed, I.VOCAB)
        torch.cuda.synchronize()


def gpu_params(P, wl):
    p = wl.params
    return P.make_params(wl.n_ranks, p["budget"], rule=p["rule"], join_mode=p["join_mode"],
                         sample_quota=p["sample_quota"], emitted_so_far=p["emitted_so_far"],
                         buffer_size=p["buffer_size"], slot_capacity=p["slot_capacity"], pad_id=p["pad_id"],
                         ignore_index=p["ignore_index"], shift_labels=p["shift_labels"])


def time_device(P, ctx, wl, din, out, steps, warmup, barrier):
    """W warm-up + K timed odb_run passes; CUDA events on the launching (current) stream.
    Returns (ms_per_step, collate_ms_avg, plan_ms_avg, post_ms_avg, launches_per_step, info)."""
    import torch

    def one():
        return P.odb_run(ctx.h, din.lengths, wl.rank_ptr, din.tokens, din.sample_ptr, din.span_ptr, din.span_lo,
                         din.span_hi, out.struct)

    info = None
    for _ in range(warmup):
        info = one()
    torch.cuda.synchronize()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = P.odb_kernel_launches(ctx.h)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(steps):
        info = one()
    ev1.record()
    torch.cuda.synchronize()
    barrier()
    ms = ev0.elapsed_time(ev1) / max(steps, 1)
    launches = (P.odb_kernel_launches(ctx.h) - l0) / max(steps, 1)
    # per-step stage events, recorded by the library on the launching stream INSIDE the timed region and read
    # here, after it (the library keeps the last 64 runs' events)
    n_read = min(steps, 64)
    stage = np.zeros(3)
    for back in range(n_read):
        stage += np.asarray(P.odb_get_timing_at(ctx.h, back))
    stage /= max(n_read, 1)
    return ms, float(stage[1]), float(stage[0]), float(stage[2]), launches, info


def time_e2e(P, ctx, wl, din, info, steps, device, device_arenas=False):
    """odb_run_host: pinned HOST inputs -> device -> whole path -> pinned HOST outputs, all inside the
    timed region (wall clock around the synchronous C call, which ends with a stream synchronize).
    device_arenas: the four arenas stay in HBM (ODB_OPT_HOST_DEVICE_ARENAS), only the tables come back."""
    import torch
    pin = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dt).pin_memory()
    h_len = pin(wl.lengths, torch.int32)
    h_sp = pin(wl.sample_ptr, torch.int64)
    h_spp = pin(wl.span_ptr, torch.int64)
    h_lo = pin(wl.span_lo if len(wl.span_lo) else np.zeros(1, np.int32), torch.int32)
    h_hi = pin(wl.span_hi if len(wl.span_hi) else np.zeros(1, np.int32), torch.int32)
    h_tok = torch.empty(wl.n_tokens + 16, dtype=torch.int32, pin_memory=True)
    h_tok.copy_(din.tokens)                      # same ids as the device buffer (untimed set-up)
    if device_arenas:
        hout = P.OutputBuffers(wl.n_ranks, 0, info.n_slots, info.samples_emitted, info.n_steps, info.samples_left, "cpu")
        dout = P.OutputBuffers(wl.n_ranks, info.total_elems, 0, 0, 0, 0, device, tables=False)
        hs, ds = hout.struct, dout.struct
        hs.d_input_ids, hs.d_labels, hs.d_position_ids = ds.d_input_ids, ds.d_labels, ds.d_position_ids
        hs.d_attention_mask, hs.arena_capacity = ds.d_attention_mask, int(info.total_elems)
    else:
        hout = P.OutputBuffers.for_plan(wl.n_ranks, info, "cpu")
    P.odb_set_option(ctx.h, P.ODB_OPT_HOST_DEVICE_ARENAS, 1 if device_arenas else 0)
    torch.cuda.synchronize()

    def one():
        return P.odb_run_host(ctx.h, h_len, wl.rank_ptr, h_tok, h_sp, h_spp, h_lo, h_hi, hout.struct)

    one()                                        # warm-up: sizes the library's device staging
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / max(steps, 1)
    h2d = (h_len.numel() * 4 + h_sp.numel() * 8 + h_spp.numel() * 8 + len(wl.span_lo) * 8 + wl.n_tokens * 4)
    E = int(info.total_elems)
    d2h = (0 if device_arenas else 13 * E) + int(info.n_slots) * (5 * 4 + 8) + (int(info.n_slots) + 1) * 8 \
        + int(info.samples_emitted) * 4 + int(info.n_steps) * 12 + (wl.n_ranks + 1) * 8 + int(info.samples_left) * 4
    P.odb_set_option(ctx.h, P.ODB_OPT_HOST_DEVICE_ARENAS, 0)
    return dt, int(h2d), int(d2h)


def check_world(args, world):
    """The printed n_gpus is the world size; it must be what --gpus asked for."""
    import torch
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if torch.cuda.device_count() < int(os.environ.get("LOCAL_RANK", "0")) + 1:
        raise SystemExit("bench.py: LOCAL_RANK %s has no CUDA device (%d visible)" % (
            os.environ.get("LOCAL_RANK", "0"), torch.cuda.device_count()))


def run_ours(args):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device. The product path has no CPU fallback.")
    import paper_2606_19989_b200 as P
    P.load()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    check_world(args, world)
    torch.cuda.set_device(local)
    device = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(device))

    def barrier():
        if world > 1:
            dist.barrier()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    wl = make_wl(args)
    din = DeviceInputs(wl, device, P)
    desc = I.describe(wl)
    result = {}
    with P.Odb(gpu_params(P, wl), max(wl.n_samples, 1), device=local) as ctx:
        P.odb_set_timing(ctx.h, True)
        if args.collate_bulk:
            P.odb_set_option(ctx.h, P.ODB_OPT_COLLATE_BULK_STORES, 1)
        info = ctx.plan(din.lengths, wl.rank_ptr)
        out = P.OutputBuffers.for_plan(wl.n_ranks, info, device)
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        ms, col_ms, plan_ms, post_ms, launches, info = time_device(P, ctx, wl, din, out, args.steps, args.warmup, barrier)
        clocks = sampler.stop() if rank == 0 else None
        ms = max_over_ranks(ms)
        col_ms_max = max_over_ranks(col_ms)
        n_samples, n_tok = int(info.samples_emitted), int(info.real_tokens)
        abytes = algorithmic_bytes(info.real_tokens, info.padded_elems)
        peak, peak_src = measured_peak()
        achieved = abytes / (col_ms_max * 1e-3) / 1e9
        wkey = cell_key(args.config, args.cv if args.config == 4 else 0, wl.params["budget"], args.rule,
                        wl.params["buffer_size"])
        traffic = ncu_traffic(wkey)
        result = {
            "metric": METRIC, "value": world * n_samples / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": workload_name(args, wl), "rule": RULE_NAMES[args.rule], "join_mode": args.join,
                       "samples": n_samples, "real_tokens": n_tok, "padded_elems": int(info.padded_elems),
                       "pad_frac": 1.0 - n_tok / max(int(info.padded_elems), 1), "n_steps": int(info.n_steps),
                       "n_slots": int(info.n_slots), "n_rounds": int(info.n_rounds),
                       "length_mean": desc["mean"], "length_cv": desc["cv"], "length_max": desc["max"],
                       "f_s": desc["f_s"],   # Pr[l < L_max / 4], the paper's short-sample fraction
                       "parallelism": "replicas only (virtual ranks live on one GPU; no inter-GPU collective)",
                       "l2": "no flush: every step reads %.1f GB of tokens and writes %.1f GB of outputs, both far "
                             "larger than the 126 MB L2" % (4 * n_tok / 1e9, 13 * int(info.padded_elems) / 1e9)},
            "tokens_per_s": world * n_tok / (ms * 1e-3),
            "hbm_gbs_whole_step": abytes / (ms * 1e-3) / 1e9,
            "stage_ms": {"planning": plan_ms, "collate_kernel": col_ms, "post": post_ms},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_over_algorithmic": traffic / abytes if traffic else None,
                         "traffic_source": ("profiles/collate_traffic.txt key %s (ncu --set full capture of this "
                                            "cell)" % wkey) if traffic else "no ncu capture of this cell",
                         "kernel": "k_collate", "algorithmic_bytes": abytes,
                         "kernel_ms": col_ms_max, "peak_source": peak_src,
                         "frac_of_nominal_8180": achieved / 8180.0},
            "gpu_launches": int(round(launches * args.steps)),
            "clocks": clocks,
        }
        result["stage_ms"]["planning_share"] = plan_ms / ms
        if not args.no_sweep and world == 1:
            # the store-side ceiling for this kernel's byte mix, and the bulk-store form of the kernel beside the adopted one
            del out
            torch.cuda.empty_cache()
            mc = mix_ceiling(P, device)
            best = max(mc["mix_stg256"], mc["mix_bulk_store"])
            result["roofline"]["mix_ceiling"] = mc
            result["roofline"]["mix_ceiling_gbs"] = best
            result["roofline"]["frac_of_mix_ceiling"] = achieved / best
            out = P.OutputBuffers.for_plan(wl.n_ranks, info, device)
            P.odb_set_option(ctx.h, P.ODB_OPT_COLLATE_BULK_STORES, 1)
            _, col_b, _, _, _, _ = time_device(P, ctx, wl, din, out, 5, 3, barrier)
            P.odb_set_option(ctx.h, P.ODB_OPT_COLLATE_BULK_STORES, 0)
            result["roofline"]["bulk_store_variant"] = {"kernel_ms": col_b, "achieved": abytes / (col_b * 1e-3) / 1e9,
                                                        "vs_adopted": col_b / col_ms_max,
                                                        "note": "k_collate<., BULK=true>: interior chunks staged in shared "
                                                                "memory, cp.async.bulk stores; not adopted unless faster"}
        if args.pipeline > 1 and world == 1:
            del out
            torch.cuda.empty_cache()
            pms = time_pipelined(P, wl, device, args.pipeline, args.steps, args.warmup)
            result["pipelined"] = {"contexts": args.pipeline, "ms_per_step": pms, "vs_single_context": pms / ms,
                                   "samples_per_s": n_samples / (pms * 1e-3),
                                   "hbm_gbs_whole_step": abytes / (pms * 1e-3) / 1e9,
                                   "whole_step_frac": abytes / (pms * 1e-3) / 1e9 / peak}
            out = P.OutputBuffers.for_plan(wl.n_ranks, info, device)
        result["launches_per_step"] = launches
        if not args.no_sweep and world == 1:
            rows = run_sweep(P, args, device, peak)
            result["sweep"] = rows
            big = [r for r in rows if r["workload"].startswith("configs[4]") and r["frac"] is not None]
            small = [r for r in rows if not r["workload"].startswith("configs[4]") and r["frac"] is not None]
            if big:
                w = min(big, key=lambda r: r["frac"])
                result["roofline"]["worst_cell"] = {"workload": w["workload"], "rule": w["rule"], "frac": w["frac"],
                                                    "whole_step_frac": w["whole_step_frac"]}
            if small:
                w = min(small, key=lambda r: r["frac"])
                result["roofline"]["worst_small_config"] = {"workload": w["workload"], "rule": w["rule"],
                                                            "frac": w["frac"], "ms_per_step": w["ms_per_step"],
                                                            "note": "sub-millisecond steps: launch latency, not HBM, bounds them"}
            result["paper_operating_point"] = paper_operating_point(P, device, peak)
            result["comparators"] = comparators(P, device)
            result["streaming"] = [streaming_output(P, device, peak, steps_per_chunk=n) for n in (40, 160)]
        # ---- e2e through the C ABI with HOST buffers (odb_run_host) -------------------------
        if not args.no_e2e:
            need = 4 * wl.n_tokens + 13 * int(info.total_elems)
            try:
                import psutil
                avail = psutil.virtual_memory().available
            except Exception:
                avail = 0
            if avail and need * 1.3 * world > avail:
                result["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                                 "note": "host RAM too small to pin %d bytes per rank" % need}
            else:
                del out
                torch.cuda.empty_cache()
                barrier()
                if args.host_staging_elems:
                    P.odb_set_option(ctx.h, P.ODB_OPT_HOST_STAGING_ELEMS, args.host_staging_elems)
                dt, h2d, d2h = time_e2e(P, ctx, wl, din, info, args.e2e_steps, device)
                dt = max_over_ranks(dt)
                result["e2e"] = {"value": world * n_samples / dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
                                 "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3, "steps": args.e2e_steps,
                                 "tokens_per_s": world * n_tok / dt, "pcie_gbs": (h2d + d2h) / dt / 1e9,
                                 "d2h_gbs": d2h / dt / 1e9, "h2d_gbs_if_alone": h2d / dt / 1e9,
                                 "device_staging": "token ring 3 x one rank, output ring 3 x %d elements (13 B each)" % (
                                     args.host_staging_elems or (1 << 25)),
                                 "api": "odb_run_host (pinned host buffers in and out)"}
                # the same call with the arenas left in HBM for a trainer on this GPU: only the inputs cross the link
                dt2, h2d2, d2h2 = time_e2e(P, ctx, wl, din, info, args.e2e_steps, device, device_arenas=True)
                dt2 = max_over_ranks(dt2)
                result["e2e_device_outputs"] = {
                    "value": world * n_samples / dt2, "unit": UNIT, "h2d_bytes_per_step": h2d2, "d2h_bytes_per_step": d2h2,
                    "ms_per_step": dt2 * 1e3, "steps": args.e2e_steps, "tokens_per_s": world * n_tok / dt2,
                    "h2d_gbs": h2d2 / dt2 / 1e9,
                    "api": "odb_run_host with ODB_OPT_HOST_DEVICE_ARENAS (pinned host inputs; arenas stay in HBM, tables "
                           "come back to the host)"}
    del din
    torch.cuda.empty_cache()
    if rank == 0 and world == 1 and not args.no_sweep:
        result["sharded_protocol_n1"] = sharded_protocol_rows()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cb, _ = cpu_baseline(args, args.cpu_sample_ranks)
        result["cpu_baseline"] = cb
    elif rank == 0:
        result["cpu_baseline"] = None
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(result), flush=True)


def run_sharded(args):
    """--shard-ranks: ONE job whose R virtual ranks are split over the N GPUs (R/N consecutive ranks per
    process), driven by the protocol of paper_2606_19989_b200/dist.py: per round one all_gather of the
    (G_r, S_r) pairs and one all_reduce of the step totals over NCCL, then the local collate and the
    all_reduce of the per-step valid-token totals.  Strong scaling: value = the job's samples / time."""
    import torch
    import torch.distributed as dist
    import paper_2606_19989_b200 as P
    from paper_2606_19989_b200 import dist as D
    P.load()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    check_world(args, world)
    torch.cuda.set_device(local)
    device = "cuda:%d" % local
    if world == 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29577")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device(device))
    else:
        dist.init_process_group("nccl", device_id=torch.device(device))
    wl_all = make_wl(args)
    if wl_all.n_ranks % world:
        raise SystemExit("--shard-ranks needs the rank count (%d) to be a multiple of --gpus" % wl_all.n_ranks)
    rl = wl_all.n_ranks // world
    wl = I.split_ranks(wl_all, world)[rank]
    t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dt).to(device)
    lengths, sample_ptr, span_ptr = t(wl.lengths, torch.int32), t(wl.sample_ptr, torch.int64), t(wl.span_ptr, torch.int64)
    z = torch.zeros(1, dtype=torch.int32, device=device)
    span_lo = t(wl.span_lo, torch.int32) if len(wl.span_lo) else z
    span_hi = t(wl.span_hi, torch.int32) if len(wl.span_hi) else z
    tokens = torch.empty(wl.n_tokens + 16, dtype=torch.int32, device=device)
    P.odb_synth_tokens(tokens, wl.token_start, wl.n_tokens, wl.token_seed, I.VOCAB)
    coll = D.TorchCollectives()
    eng = D.CudaEngine(gpu_params(P, wl), max(wl.n_samples, 1), lengths, wl.rank_ptr, device=local)
    P.odb_set_timing(eng.ctx.h, True)
    batched = not args.per_round_exchange
    info, _ = D.run(D.plan_protocol(eng, wl_all.n_ranks, rank * rl, batched=batched), coll, device)
    out = P.OutputBuffers.for_plan(rl, info, device)

    def one():
        info, _ = D.run(D.plan_protocol(eng, wl_all.n_ranks, rank * rl, batched=batched), coll, device)
        eng.collate(tokens, sample_ptr, span_ptr, span_lo, span_hi, out)
        D.run(D.step_valid_protocol(out.table("step_valid_tokens")), coll, device)
        return info

    for _ in range(args.warmup):
        one()
    torch.cuda.synchronize()
    dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = P.odb_kernel_launches(eng.ctx.h)
    col = 0.0
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        info = one()
    ev1.record()
    torch.cuda.synchronize()
    dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = P.odb_kernel_launches(eng.ctx.h) - l0
    # the collate kernel's time, read AFTER the timed region (odb_get_timing waits for the stage events): two more steps
    for _ in range(2):
        one()
        col += P.odb_get_timing(eng.ctx.h)[1] * args.steps / 2.0
    tt = torch.tensor([ev0.elapsed_time(ev1) / max(args.steps, 1), col / max(args.steps, 1)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ms, col_ms = float(tt[0]), float(tt[1])
    tot = torch.tensor([int(info.samples_emitted), int(info.real_tokens), int(info.padded_elems)], dtype=torch.int64, device=device)
    loc = tot.clone()
    dist.all_reduce(tot)
    n_samples, n_tok, n_pad = (int(x) for x in tot.tolist())
    peak, peak_src = measured_peak()
    ab_local = algorithmic_bytes(int(loc[1]), int(loc[2]))
    achieved = ab_local / (col_ms * 1e-3) / 1e9
    eng.close()
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": n_samples / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "int32", "data": "synthetic",
            "config": {"workload": workload_name(args, wl_all), "rule": RULE_NAMES[args.rule], "join_mode": args.join,
                       "samples": n_samples, "real_tokens": n_tok, "padded_elems": n_pad, "n_steps": int(info.n_steps),
                       "n_rounds": int(info.n_rounds),
                       "parallelism": "virtual ranks sharded over %d GPU(s), %d per GPU; %s over NCCL" % (
                           world, rl, "batched exchange: all_gather(n_r), all_gather(G tables), all_reduce(step totals) "
                           "for every round without leftovers, then per round all_gather(G,S) + all_reduce" if batched
                           else "per round all_gather(G,S) + all_reduce(step totals)"),
                       "l2": "no flush: inputs and outputs are far larger than the 126 MB L2"},
            "tokens_per_s": n_tok / (ms * 1e-3), "stage_ms": {"collate_kernel": col_ms},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "kernel": "k_collate (rank 0's share)", "algorithmic_bytes": ab_local,
                         "kernel_ms": col_ms, "peak_source": peak_src},
            "gpu_launches": int(launches), "clocks": clocks, "e2e": None, "cpu_baseline": None}), flush=True)


def time_pipelined(P, wl, device, n_ctx, steps, warmup):
    """n_ctx contexts (own scratch, own outputs, own stream), the same resident inputs, odb_run called round-robin:
    while one context's collate kernel runs, the next context's planning kernels are already enqueued on another
    stream (odb_run returns as soon as the plan sizes are known).  Device time per step over all contexts."""
    import torch
    local = int(device.split(":")[1])
    din = DeviceInputs(wl, device, P)
    ctxs, outs, streams = [], [], []
    try:
        for i in range(n_ctx):
            c = P.Odb(gpu_params(P, wl), max(wl.n_samples, 1), device=local)
            info = c.plan(din.lengths, wl.rank_ptr)
            ctxs.append(c)
            outs.append(P.OutputBuffers.for_plan(wl.n_ranks, info, device))
            streams.append(torch.cuda.Stream(device=device))
        torch.cuda.synchronize()

        def one(i):
            with torch.cuda.stream(streams[i]):
                return P.odb_run(ctxs[i].h, din.lengths, wl.rank_ptr, din.tokens, din.sample_ptr, din.span_ptr, din.span_lo,
                                 din.span_hi, outs[i].struct, stream=streams[i])

        for k in range(warmup * n_ctx):
            one(k % n_ctx)
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for s_ in streams:
            s_.wait_event(ev0)
        for k in range(steps * n_ctx):
            one(k % n_ctx)
        cur = torch.cuda.current_stream()
        for s_ in streams:
            cur.wait_stream(s_)
        ev1.record()
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / (steps * n_ctx)
    finally:
        for c in ctxs:
            c.close()
        del outs, din
        torch.cuda.empty_cache()


def mix_ceiling(P, device, n_elems=1 << 29):
    """What the collate kernel's byte mix (4 B read + 13 B written per element) reaches with trivial indexing on this
    device, in the two store forms the kernel can use, next to a pure-store stream and a copy (odb_probe_bandwidth)."""
    import torch
    src = torch.empty(n_elems, dtype=torch.int32, device=device)
    o = [torch.empty(n_elems, dtype=torch.int32, device=device) for _ in range(3)]
    m = torch.empty(n_elems, dtype=torch.uint8, device=device)
    src.zero_()
    names = {0: "mix_stg256", 1: "mix_bulk_store", 2: "store_only_stg256", 3: "store_only_bulk_store", 4: "copy_4r_4w"}
    bytes_per = {0: 17, 1: 17, 2: 13, 3: 13, 4: 8}
    out = {"n_elems": n_elems, "unit": "GB/s"}
    for kind, name in names.items():
        ms = P.odb_probe_bandwidth(kind, src, o[0], o[1], o[2], m, n_elems, reps=5)
        out[name] = bytes_per[kind] * n_elems / (ms * 1e-3) / 1e9
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    o[0].zero_()
    ev0.record()
    for _ in range(5):
        o[0].zero_()
    ev1.record()
    torch.cuda.synchronize()
    out["memset_torch_zero"] = 5 * 4 * n_elems / (ev0.elapsed_time(ev1) * 1e-3) / 1e9
    del src, o, m
    torch.cuda.empty_cache()
    return out


def comparators(P, device):
    """Shape statistics of ODB beside the paper's offline comparators as planners (F4: GMT / BMT; HFG)
    on the synthetic configs: samples per update (global), padding fraction, steps -- the quantities of the paper's
    Tables 13 / 14.  Planning only (lengths; no token is touched).  The offline planners see the pooled
    lengths of all ranks; HFG's fixed batch size is the largest one whose padded area fits the budget for the longest
    sample (its "full-epoch-safe" batch size), its megabatch = 50 batches per rank (the HuggingFace default),
    BMT buckets hold 4096 samples."""
    import torch
    local = int(device.split(":")[1])
    rows = []
    for idx in (1, 2, 3):
        wl = I.make_workload(idx)
        W, N, budget = wl.n_ranks, wl.n_samples, wl.params["budget"]
        d_len = torch.from_numpy(wl.lengths).to(device)
        rng = np.random.default_rng(600 + idx)
        d_perm = torch.from_numpy(rng.permutation(N).astype(np.int32)).to(device)
        d_key = torch.from_numpy(rng.integers(0, 2**31 - 1, N).astype(np.int32)).to(device)
        bs = max(1, budget // int(wl.lengths.max()))

        def row(method, info, ms):
            rows.append({"workload": "configs[%d] %s" % (idx, I.bj_config(idx)["name"]), "method": method,
                         "samples_per_update": int(info.samples_emitted) / max(int(info.n_steps), 1),
                         "real_tokens_per_update": int(info.real_tokens) / max(int(info.n_steps), 1),
                         "pad_frac": 1.0 - int(info.real_tokens) / max(int(info.padded_elems), 1),
                         "n_steps": int(info.n_steps), "samples_emitted": int(info.samples_emitted), "plan_ms": ms})

        def timed(fn):
            fn()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            info = fn()
            torch.cuda.synchronize()
            return info, (time.perf_counter() - t0) * 1e3

        with P.Odb(gpu_params(P, wl), N, device=local) as ctx:
            info, ms = timed(lambda: ctx.plan(d_len, wl.rank_ptr))
            row("ODB (rule THRESHOLD, whole-stream window)", info, ms)
        wl1k = I.make_workload(idx)
        wl1k.params["buffer_size"] = 1024
        with P.Odb(gpu_params(P, wl1k), N, device=local) as ctx:
            info, ms = timed(lambda: ctx.plan(d_len, wl.rank_ptr))
            row("ODB (rule THRESHOLD, buffer 1024)", info, ms)
        prm = P.make_params(W, budget, rule=P.ODB_RULE_MAXFIT_ASC)
        for name, planner, kw in (("GMT-oracle", P.ODB_PLANNER_GMT, {}),
                                  ("BMT-oracle (bucket 4096)", P.ODB_PLANNER_BMT, dict(d_perm=d_perm, d_shuffle_key=d_key, size=4096)),
                                  ("HFG-oracle (bs %d, megabatch %d)" % (bs, bs * W * 50), P.ODB_PLANNER_HFG,
                                   dict(d_perm=d_perm, size=bs * W * 50, batch_size=bs))):
            with P.Odb(prm, N, device=local) as ctx:
                def fn():
                    P.odb_offline_plan(ctx.h, planner, d_len, N, **kw)
                    return P.odb_plan_query(ctx.h)
                info, ms = timed(fn)
                row(name, info, ms)
    return rows


def cell_key(config, cv, budget, rule, buffer_size=0):
    k = "config%d_cv%g_L%d_rule%d" % (config, cv, budget, rule)
    return k + ("_buf%d" % buffer_size if buffer_size else "")


def measure_workload(P, wl, device, steps, warmup, options=None):
    """One workload through odb_run on `device` (own context, inputs and outputs); returns a row dict."""
    import torch
    din = DeviceInputs(wl, device, P)
    with P.Odb(gpu_params(P, wl), max(wl.n_samples, 1), device=int(device.split(":")[1])) as ctx:
        for opt, val in (options or {}).items():
            P.odb_set_option(ctx.h, opt, val)
        P.odb_set_timing(ctx.h, True)
        info = ctx.plan(din.lengths, wl.rank_ptr)
        out = P.OutputBuffers.for_plan(wl.n_ranks, info, device)
        ms, col_ms, plan_ms, post_ms, launches, info = time_device(P, ctx, wl, din, out, steps, warmup, lambda: None)
        del out
    del din
    torch.cuda.empty_cache()
    ab = algorithmic_bytes(info.real_tokens, info.padded_elems)
    n_rounds = int(info.n_rounds)
    return {"rule": RULE_NAMES[wl.params["rule"]], "join_mode": wl.params["join_mode"],
            "buffer_size": wl.params["buffer_size"], "ms_per_step": ms,
            "samples_per_s": int(info.samples_emitted) / (ms * 1e-3),
            "tokens_per_s": int(info.real_tokens) / (ms * 1e-3),
            "planning_ms": plan_ms, "collate_ms": col_ms, "post_ms": post_ms,
            "planning_share": plan_ms / max(ms, 1e-9), "collate_gbs": ab / (col_ms * 1e-3) / 1e9 if col_ms > 0 else None,
            "whole_step_gbs": ab / (ms * 1e-3) / 1e9, "algorithmic_bytes": ab,
            "n_steps": int(info.n_steps), "n_rounds": n_rounds, "launches_per_step": launches,
            "planning_ms_per_round": plan_ms / max(n_rounds, 1),
            "pad_frac": 1.0 - int(info.real_tokens) / max(int(info.padded_elems), 1)}


def run_sweep(P, args, device, peak):
    """The nine (CV, budget) cells of configs[4] (rule THRESHOLD; --sweep adds MAXFIT_ASC) and configs[1..3]
    (configs[3] in join and non-join mode): per-row collate fraction of the measured peak."""
    rows = []
    rules = (0, 1) if args.sweep else (0,)

    def add(name, key, wl):
        row = measure_workload(P, wl, device, 5, 3)
        row["workload"] = name
        row["frac"] = row["collate_gbs"] / peak if row["collate_gbs"] else None
        row["whole_step_frac"] = row["whole_step_gbs"] / peak
        row["traffic"] = ncu_traffic(key)
        rows.append(row)

    for cv, L in I.config5_cells():
        for rule in rules:
            add("configs[4] CV %g L %d" % (cv, L), cell_key(4, cv, L, rule), I.make_workload(4, cv=cv, budget=L, rule=rule))
    for idx in (1, 2, 3):
        c = I.bj_config(idx)
        for rule in rules:
            add("configs[%d] %s" % (idx, c["name"]), cell_key(idx, 0, c["budget"], rule), I.make_workload(idx, rule=rule))
    add("configs[3] highcv_longtail non-join (quota)", "config3_nonjoin", I.make_workload(3, join_mode=0))
    return rows


def paper_operating_point(P, device, peak):
    """The paper's operating point: a 1024-sample grouping buffer per rank, i.e. tens of protocol rounds
    per rank stream, on the configs[4] recipe (CV 1.0, budget 65536)."""
    wl = I.make_workload(4, cv=1.0, budget=65536)
    wl.params["buffer_size"] = 1024
    row = measure_workload(P, wl, device, 5, 3)
    row["workload"] = "configs[4] CV 1 L 65536, buffer_size 1024 (P:28)"
    row["frac"] = row["collate_gbs"] / peak if row["collate_gbs"] else None
    row["whole_step_frac"] = row["whole_step_gbs"] / peak
    row["traffic"] = ncu_traffic(cell_key(4, 1.0, 65536, 0, 1024))
    row["planner"] = "round-parallel (k_spec_form / k_spec_commit; k_rounds resumes at the first round that overflows)"
    # the same job with every round in the sequential device-side loop (ODB_OPT_ROUND_PARALLEL = 0)
    seq = measure_workload(P, wl, device, 5, 3, options={P.ODB_OPT_ROUND_PARALLEL: 0})
    row["sequential_round_loop"] = {k: seq[k] for k in ("ms_per_step", "planning_ms", "planning_ms_per_round",
                                                        "launches_per_step")}
    return row


def sharded_protocol_rows(steps=5, warmup=3):
    """The multi-process protocol (F1: paper_2606_19989_b200/dist.py over NCCL) at the paper's operating point, on this
    one GPU (world size 1 -- no N > 1 number can be taken here): the batched exchange beside one exchange per round.
    Each row is a `bench.py --shard-ranks` run in a process of its own (its own NCCL world); a failure is reported,
    it never breaks the main line."""
    import socket
    import subprocess
    rows = []
    for name, extra in (("batched exchange (J rounds: 3 collectives + 2 scalar exchanges)", []),
                        ("one exchange per round (P:52)", ["--per-round-exchange"])):
        sk = socket.socket()
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
        sk.close()
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "LOCAL_WORLD_SIZE"):
            env.pop(k, None)
        cmd = [sys.executable, os.path.abspath(__file__), "--shard-ranks", "--buffer-size", "1024", "--steps", str(steps),
               "--warmup", str(warmup)] + extra
        try:
            r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=240)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            rows.append({"exchange": name, "ms_per_step": d["ms_per_step"], "samples_per_s": d["value"],
                         "collate_ms": d["stage_ms"]["collate_kernel"], "gpu_launches_per_step": d["gpu_launches"] / steps,
                         "n_rounds": d["config"]["n_rounds"], "n_gpus": d["n_gpus"]})
        except Exception as e:  # noqa: BLE001 (a measurement beside the line, never the line itself)
            rows.append({"exchange": name, "error": repr(e)[:200]})
    return rows


def streaming_output(P, device, peak, steps_per_chunk=40, reps=5):
    """The paper's operating point (buffer 1024) with STREAMING output: odb_plan, then the plan's steps pulled
    `steps_per_chunk` at a time (about one protocol round) through two bounded output buffers on two streams
    (odb_collate_steps; what StepStream does).  Wall clock around the host calls with a device synchronise on both
    sides: time to the first chunk, and the whole pass beside the one-launch odb_run of the same job."""
    import torch
    wl = I.make_workload(4, cv=1.0, budget=65536)
    wl.params["buffer_size"] = 1024
    din = DeviceInputs(wl, device, P)
    inputs = (din.tokens, din.sample_ptr, din.span_ptr, din.span_lo, din.span_hi)
    R = wl.n_ranks
    slot_elems = (max(int(wl.params["budget"]), int(wl.lengths.max())) + 15) // 16 * 16
    with P.Odb(gpu_params(P, wl), wl.n_samples, device=int(device.split(":")[1])) as ctx:
        info = P.odb_plan(ctx.h, din.lengths, wl.rank_ptr)
        K = int(info.n_steps)
        slots = R * steps_per_chunk
        bufs = [P.OutputBuffers(R, slots * slot_elems, slots, wl.n_samples, steps_per_chunk, 0, device) for _ in range(2)]
        streams = [torch.cuda.Stream(device=device) for _ in range(2)]
        n_chunks = (K + steps_per_chunk - 1) // steps_per_chunk

        def one_pass(first_only=False):
            P.odb_plan(ctx.h, din.lengths, wl.rank_ptr)
            elems = 0
            for i in range(n_chunks):
                lo = i * steps_per_chunk
                ci = P.odb_collate_steps(ctx.h, lo, min(K, lo + steps_per_chunk), *inputs, bufs[i & 1].struct,
                                         stream=streams[i & 1].cuda_stream)
                elems = max(elems, int(ci.total_elems))
                if first_only:
                    break
            return elems

        one_pass()
        torch.cuda.synchronize()
        l0 = P.odb_kernel_launches(ctx.h)
        t0 = time.perf_counter()
        for _ in range(reps):
            chunk_elems = one_pass()
        torch.cuda.synchronize()
        ms = (time.perf_counter() - t0) / reps * 1e3
        launches = (P.odb_kernel_launches(ctx.h) - l0) / reps
        t0 = time.perf_counter()
        for _ in range(reps):
            one_pass(first_only=True)
            torch.cuda.synchronize()
        first_ms = (time.perf_counter() - t0) / reps * 1e3
        del bufs
    del din
    torch.cuda.empty_cache()
    ab = algorithmic_bytes(info.real_tokens, info.padded_elems)
    return {"workload": "configs[4] CV 1 L 65536, buffer_size 1024 (P:28)", "api": "odb_plan + odb_collate_steps",
            "steps_per_chunk": steps_per_chunk, "chunks": n_chunks, "ms_per_pass": ms,
            "samples_per_s": int(info.samples_emitted) / (ms * 1e-3), "whole_pass_gbs": ab / (ms * 1e-3) / 1e9,
            "whole_pass_frac": ab / (ms * 1e-3) / 1e9 / peak, "ms_to_first_chunk": first_ms,
            "launches_per_pass": launches, "largest_chunk_bytes": 13 * chunk_elems,
            "output_buffer_bytes": 2 * 13 * R * steps_per_chunk * slot_elems,
            "whole_plan_output_bytes": 13 * int(info.total_elems),
            "timing": "wall clock around the host calls, device synchronised on both sides"}


# --------------------------------------------------------------------------------------------
# --gpus N without torchrun: start the N processes ourselves
# --------------------------------------------------------------------------------------------
def launcher_envs(n, port, base_env):
    """Environment of each of the n worker processes (rank i on GPU i, rendezvous on 127.0.0.1)."""
    envs = []
    for i in range(n):
        e = dict(base_env)
        e.update(RANK=str(i), LOCAL_RANK=str(i), WORLD_SIZE=str(n), LOCAL_WORLD_SIZE=str(n),
                 MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        e.setdefault("NCCL_DEBUG", "INFO")            # communicator lines (rank counts) stay visible in stderr
        e.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        envs.append(e)
    return envs


def free_port():
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def self_launch(args):
    """One process per GPU; rank 0 prints the JSON line on our stdout.  Exits non-zero when the box has fewer
    than --gpus CUDA devices (never a silent N=1 number)."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        sys.stderr.write("bench.py: --gpus %d but this box has %d CUDA device(s); refusing to report an N=%d number "
                         "from fewer GPUs\n" % (args.gpus, have, args.gpus))
        sys.exit(2)
    envs = launcher_envs(args.gpus, free_port(), os.environ)
    procs = [subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=e,
                              stdout=(None if i == 0 else subprocess.DEVNULL)) for i, e in enumerate(envs)]
    rcs = [p.wait() for p in procs]
    sys.exit(max(abs(rc) for rc in rcs))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)       # rank 0 alone runs it, whatever --gpus says
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        self_launch(args)
    elif args.shard_ranks:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
