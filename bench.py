#!/usr/bin/env python
"""bench.py -- regular-force pair interactions/s at N = 1M (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n-i 8192] [--no-sweep] [--impl reference]

A "step" is one pass of the whole hot path over BASELINE.json config 4
(N = 1,048,576 Plummer + Kroupa IMF + 5 % binaries, synthetic, seed 0):
    nb_set_j (ingest + re-layout)  ->  nb_predict_all(t)  ->  nb_regular(active block of n_i)
`value` counts n_i * N pair interactions per step with all inputs resident in HBM; `e2e` runs the same
step through the HOST-pointer C-ABI calls (pinned host buffers, copies inside the timed region).
Under torchrun each rank holds all N j-particles and takes its shard of a world_size * n_i active
block (i-sharding = the paper's copy algorithm; no data-path collective) -> "scaling": "weak".

--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same
workload; it is the only leg besides cpu_baseline that executes anything under oracle/.
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
sys.path.insert(0, ROOT)

FLOP_PER_INTERACTION = 60.0          # BASELINE.json north_star convention (force + jerk)
METRIC = "regular-force pair interactions/s at N=1M"
UNIT = "pair interactions/s"
WORKLOAD = "cfg4_plummer1m_kroupa_bin5_headline"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--n-i", type=int, default=8192, help="active-block size per GPU")
    ap.add_argument("--N", type=int, default=1048576, help="override N (debug only; the metric is N=1M)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--variant", type=int, default=-1, help="force a force-kernel variant (tuning experiments)")
    ap.add_argument("--shard", default="i", choices=["i", "j"],
                    help="N > 1 ranks: i = every rank holds all N bodies and takes its share of a world x n_i block (no "
                         "collective, weak scaling; default); j = every rank holds N / world bodies and all ranks evaluate "
                         "the SAME n_i block (SURVEY 8(f) NEXT-4: state all-reduce, sums / lists all-gather; strong scaling)")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the NEXT-row timings (nb_block_step, nb_irregular, ...)")
    ap.add_argument("--headline-only", action="store_true",
                    help="skip the sweeps of BASELINE.json configs 3 (N=262144) and 5 (King core, overflowing rows), "
                         "which run by default")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# ----------------------------------------------------------------------------- helpers

class ClockSampler:
    """Samples SM clocks / throttle reasons with nvidia-smi DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, mx = float(f[0]), float(f[1])
            except ValueError:
                continue
            if t0 - 0.05 <= ts <= t1 + 0.15:
                sm.append(clk); smax.append(mx)
                try:
                    power.append(float(f[2]))
                except ValueError:
                    pass
                for nme, val in zip(names, f[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nme)
        if not sm:      # region shorter than the sampling period: take the nearest samples
            for ts, line in self.rows[-3:]:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0])); smax.append(float(f[1]))
                except (ValueError, IndexError):
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def build_workload(N: int, n_total: int):
    import nbgen
    cfg = nbgen.make_config(4, N=N)
    idx, h2 = nbgen.active_block(cfg, min(n_total, N))
    return cfg, idx, h2


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return p, "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


# ----------------------------------------------------------------------------- reference arm (CPU oracle)

def cpu_oracle_rate(cfg, idx, h2, seconds_target=12.0, fixed_n=None):
    """Oracle (as it stands) on a bounded sample: the first n of the active block against all N."""
    import oracle
    oracle.build()
    threads = oracle.num_threads()
    N = cfg["N"]
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    if fixed_n is None:
        probe = min(len(idx), 2 * threads)
        t = time.perf_counter()
        oracle.regular(cfg["m"], xp, vp, idx[:probe], h2[:probe], cfg["cap"])
        dt = time.perf_counter() - t
        n = int(min(len(idx), max(probe, seconds_target / max(dt, 1e-6) * probe)))
        n = max(threads, n // threads * threads)
    else:
        n = fixed_n
    t = time.perf_counter()
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    oracle.regular(cfg["m"], xp, vp, idx[:n], h2[:n], cfg["cap"])
    dt = time.perf_counter() - t
    return dict(value=n * N / dt, unit=UNIT, cores=threads, kind="oracle",
                sample=f"predict_all + first {n} of the {len(idx)}-particle active block x all N={N} j "
                       f"({n * N:.3e} pairs, {dt:.1f} s, FP64 direct sum, OpenMP over i)", n_sample=n, seconds=dt)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, idx, h2 = build_workload(args.N, args.n_i)
    import oracle
    oracle.build()
    threads = oracle.num_threads()
    # bound the whole run (warmup + steps) to a few minutes: ~6 s of CPU work per step
    first = cpu_oracle_rate(cfg, idx, h2, seconds_target=6.0)
    n = first["n_sample"]
    for _ in range(max(args.warmup - 1, 0)):
        cpu_oracle_rate(cfg, idx, h2, fixed_n=n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        cpu_oracle_rate(cfg, idx, h2, fixed_n=n)
    dt = time.perf_counter() - t0
    value = args.steps * n * cfg["N"] / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "N": cfg["N"], "n_i": int(args.n_i), "sample_n_i": n,
                   "note": "CPU oracle (oracle/nbody_oracle.c) on the host cores; each step = predict_all + a bounded "
                           "sample of the active block against all N"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"first {n} of {args.n_i} active particles x N={cfg['N']} per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- B200 arm

def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_1504_03687_b200 as nb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the B200 arm has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()

    import nbgen
    N = args.N
    if args.shard == "j":
        return run_b200_jsharded(args, world, rank, local)
    cfg, idx_all, h2_all = build_workload(N, args.n_i * world)
    idx_np, h2_np = nbgen.shard_active_block(idx_all, h2_all, rank, world)   # i-sharding, no collective
    n_i = int(idx_np.shape[0])
    cap = cfg["cap"]

    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()
    ctx = nb.nb_open(N, cap, stream)
    f64 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
    jstate = [f64(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")]
    idx = torch.from_numpy(np.ascontiguousarray(idx_np)).to(dev)
    h2 = f64(h2_np)
    out = dict(acc=torch.empty((n_i, 3), dtype=torch.float64, device=dev),
               jerk=torch.empty((n_i, 3), dtype=torch.float64, device=dev),
               pot=torch.empty(n_i, dtype=torch.float64, device=dev),
               nnb=torch.empty(n_i, dtype=torch.int32, device=dev),
               nblist=torch.empty((n_i, cap), dtype=torch.int32, device=dev),
               overflow=torch.empty(n_i, dtype=torch.int32, device=dev))
    t_pred = float(cfg["t"])
    if args.variant >= 0:
        ctx.tune("force_variant", args.variant)

    def step():
        ctx.set_j(*jstate)              # a1
        ctx.predict_all(t_pred)         # a2
        ctx.regular(idx, h2, **out)     # a3-a7

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, CUDA events on the context's stream, barrier + sync on both sides
    ctx.tune("profile", 1)
    launches0 = ctx.info("kernel_launches")
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    w0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize(); barrier()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(w0, w1) if sampler else None
    launches = ctx.info("kernel_launches") - launches0
    plan = {"variant": ctx.info("last_variant"), "jsplit": ctx.info("last_jsplit"), "grid": ctx.info("last_grid")}
    force_ns = ctx.info("force_kernel_ns")
    force_cnt = ctx.info("force_kernel_count")
    ctx.tune("profile", 0)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
        tl = torch.tensor([launches], dtype=torch.int64, device=dev)
        dist.all_reduce(tl, op=dist.ReduceOp.SUM)
        launches = int(tl.item())
    pairs_per_step = float(n_i) * N * world
    value = pairs_per_step * args.steps / (ms * 1e-3)

    # ---- e2e: same step through the HOST-pointer ABI (pinned buffers; copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hj = [pin(np.asarray(cfg[k], dtype=np.float64)) for k in ("m", "x0", "v0", "a0", "j0", "t0")]
        hidx, hh2 = pin(idx_np), pin(np.asarray(h2_np, dtype=np.float64))
        hout = dict(acc=torch.empty((n_i, 3), dtype=torch.float64).pin_memory(),
                    jerk=torch.empty((n_i, 3), dtype=torch.float64).pin_memory(),
                    pot=torch.empty(n_i, dtype=torch.float64).pin_memory(),
                    nnb=torch.empty(n_i, dtype=torch.int32).pin_memory(),
                    nblist=torch.empty((n_i, cap), dtype=torch.int32).pin_memory(),
                    overflow=torch.empty(n_i, dtype=torch.int32).pin_memory())

        def step_host():        # one C-ABI call: chunked H2D behind the force launches, results in host memory
            ctx.step_host(*hj, t_pred, hidx, hh2, **hout)

        def step_host_separate():   # the same step as three calls, nothing overlapped (context for the number above)
            ctx.set_j_host(*hj)
            ctx.predict_all(t_pred)
            ctx.regular_host(hidx, hh2, **hout)

        def time_host(fn, ke):
            for _ in range(2):
                fn()
            barrier(); torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(ke):
                fn()
            e1.record(stream)
            torch.cuda.synchronize(); barrier()
            wall = time.perf_counter() - t0
            ms_e = max(e0.elapsed_time(e1), wall * 1e3)     # host-blocking calls: wall clock bounds it
            if world > 1:
                t = torch.tensor([ms_e], dtype=torch.float64, device=dev)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                ms_e = float(t.item())
            return ms_e

        ke = max(3, min(args.steps, 10))
        l0 = ctx.info("kernel_launches")
        ms_e = time_host(step_host, ke)
        e2e_launches = (ctx.info("kernel_launches") - l0) // (ke + 2)
        ms_sep = time_host(step_host_separate, ke)
        h2d = 14 * N * 8 + n_i * (4 + 8) + 14 * n_i * 8
        maxc = int(hout["nnb"].clamp(max=cap).max())        # list columns copied back: those some row uses
        d2h = n_i * (7 * 8 + 4 + 4) + n_i * maxc * 4
        e2e = {"value": pairs_per_step * ke / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "list_columns_copied": maxc, "steps": ke, "ms_per_step": ms_e / ke,
               "call": "nb_step_host (j-state sent in 5 chunks on a copy stream, force launches behind them)",
               "gpu_launches_per_step": int(e2e_launches),
               "separate_calls": {"value": pairs_per_step * ke / (ms_sep * 1e-3), "ms_per_step": ms_sep / ke,
                                  "call": "nb_set_j_host + nb_predict_all + nb_regular_host"},
               "checksum_pot": float(hout["pot"].sum())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (force_kernel): plain FP32 issue -> "alu"
    pk, pk_src = peaks()
    sm_count = ctx.info("sm_count")
    sm_max_mhz = float((clocks or {}).get("sm_max_mhz") or pk.get("sm_max_mhz", 1965.0))
    peak_tflops = sm_count * 128 * 2 * sm_max_mhz * 1e6 / 1e12
    force_ms = force_ns / max(force_cnt, 1) * 1e-6
    ach_tflops = FLOP_PER_INTERACTION * float(n_i) * N / (force_ms * 1e-3) / 1e12
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch: from the committed `ncu --set full` captures
    # (profiles/force_kernel_traffic.csv, one row per captured launch); the row must match the timed launch
    # (n_i, N, kernel variant, j-splits) -- otherwise null, never a stale constant
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "force_kernel_traffic.csv")
    if os.path.exists(tpath):
        import csv
        with open(tpath) as f:
            for row in csv.DictReader(f):
                if (int(row["n_i"]) == n_i and int(row["N"]) == N and int(row.get("variant", -1)) == plan["variant"]
                        and int(row.get("jsplit", -1)) == plan["jsplit"]):
                    traffic = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
                    traffic_src = row["source"]
    roofline = {
        "bound": "alu", "kernel": "nbreg::force_kernel", "achieved": ach_tflops, "peak": peak_tflops,
        "unit": "TFLOP/s", "frac": ach_tflops / peak_tflops, "traffic": traffic, "traffic_source": traffic_src,
        "algorithmic_bytes": 40 * N,
        "flop_per_interaction": FLOP_PER_INTERACTION, "avg_launch_ms": force_ms, "launches_timed": int(force_cnt),
        "interactions_per_launch": float(n_i) * N,
        "peak_how": f"{sm_count} SMs x 128 FP32 lanes x 2 flop x {sm_max_mhz:.0f} MHz (max SM clock; DESIGN.md)",
        "frac_at_sampled_clock": (ach_tflops / (sm_count * 128 * 2 * clocks["sm_mhz"] * 1e6 / 1e12)
                                  if clocks and clocks.get("sm_mhz") else None),
        "share_of_step": force_ms / (ms / args.steps),
    }

    # ---- sweep vs block size (the metric is "vs block size"): nb_regular alone and predict_all + regular,
    #      3 warm-ups, 10 timed repeats each, median and min (SURVEY 8(d) timing protocol)
    def sweep_config(sctx, scfg, sizes, sN):
        rows = []
        st_pred = float(scfg["t"])
        for n in sizes:
            if n > sN:
                continue
            si, sh = nbgen.active_block(scfg, n)
            si_d, sh_d = torch.from_numpy(si).to(dev), f64(sh)
            # (1) nb_regular alone, the predicted records resident (the metric); (2) the block cost
            # nb_predict_all + nb_regular in the default mode, where a block of <= 128 particles predicts
            # inside the force kernel (NB_TUNE_FUSE_PREDICT)
            sctx.tune("fuse_predict", 0)
            sctx.predict_all(st_pred)
            so = sctx.regular_alloc(si_d, sh_d)
            for _ in range(2):
                sctx.regular(si_d, sh_d, **so)
            torch.cuda.synchronize()
            t_reg, t_blk = [], []
            for _ in range(10):
                a, b = (torch.cuda.Event(enable_timing=True) for _ in range(2))
                a.record(stream); sctx.regular(si_d, sh_d, **so); b.record(stream)
                torch.cuda.synchronize()
                t_reg.append(a.elapsed_time(b))
            sctx.tune("fuse_predict", 1)
            for rep_ in range(13):
                a, b = (torch.cuda.Event(enable_timing=True) for _ in range(2))
                a.record(stream); sctx.predict_all(st_pred); sctx.regular(si_d, sh_d, **so); b.record(stream)
                torch.cuda.synchronize()
                if rep_ >= 3:
                    t_blk.append(a.elapsed_time(b))
            # the same block cost back to back in the stream (what a block loop sees: no idle-to-launch latency)
            a, b = (torch.cuda.Event(enable_timing=True) for _ in range(2))
            n_stream = 20 if n <= 4096 else 4
            a.record(stream)
            for _ in range(n_stream):
                sctx.predict_all(st_pred); sctx.regular(si_d, sh_d, **so)
            b.record(stream)
            torch.cuda.synchronize()
            t_stream = a.elapsed_time(b) / n_stream
            sctx.tune("stats", 1)                         # how many warps differenced in their local frame
            sctx.regular(si_d, sh_d, **so)
            lw, tw = sctx.info("local_warps"), sctx.info("total_warps")
            sctx.tune("stats", 0)
            best, med = min(t_reg), float(np.median(t_reg))
            rate = float(n) * sN / (best * 1e-3)
            rows.append({"n_i": n, "ms": best, "ms_median": med, "ms_predict_plus_regular": float(np.median(t_blk)),
                         "ms_predict_plus_regular_in_stream": t_stream,
                         "pairs_per_s": rate, "frac_fp32_peak": rate * FLOP_PER_INTERACTION / 1e12 / peak_tflops,
                         "variant": sctx.info("last_variant"), "jsplit": sctx.info("last_jsplit"),
                         "fused_predict": sctx.info("last_fused"), "reordered": sctx.info("last_reordered"),
                         "local_frame_warp_frac": lw / max(tw, 1),
                         "overflow_rows": int(so["overflow"].sum()), "nnb_mean": float(so["nnb"].float().mean())})
            del so
        return rows

    sweep = None
    if not args.no_sweep and world == 1:
        sweep = sweep_config(ctx, cfg, [8, 16, 32] + list(cfg["sweep"]), N)   # 8, 16, 32: the j-packed tiny-block variants
    other = None
    if not args.headline_only and not args.no_sweep and world == 1 and N == 1048576:
        other = {}
        for kcfg in (3, 5):
            ocfg = nbgen.make_config(kcfg)
            octx = nb.nb_open(ocfg["N"], ocfg["cap"], stream)
            octx.set_j(*[f64(ocfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")])
            octx.predict_all(float(ocfg["t"]))
            other[ocfg["name"]] = {"N": ocfg["N"], "nb_cap": ocfg["cap"], "sweep": sweep_config(octx, ocfg, ocfg["sweep"], ocfg["N"])}
            octx.close()

    # ---- the steps either side of the path, timed alone; not part of `value`
    extras = None
    if not args.no_extras and world == 1:
        def timed(fn, reps=5):
            best = 1e30
            for _ in range(reps):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); fn(); b.record(stream)
                torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b))
            return best
        ctx.regular(idx, h2, **out)                      # lists of the timed block
        torch.cuda.synchronize()
        nn = int(out["nnb"].clamp(max=cap).sum())
        irr = dict(acc=torch.empty_like(out["acc"]), jerk=torch.empty_like(out["jerk"]), pot=torch.empty_like(out["pot"]))
        ms_irr = timed(lambda: ctx.irregular(t_pred, idx, out["nnb"], out["nblist"], **irr))
        sub = [t[idx.long()].contiguous() for t in jstate]
        ms_upd = timed(lambda: ctx.update_j(idx, *sub))
        ctx.tune("fuse_predict", 0)                      # launch the predictor kernel at once: timed alone
        ctx.predict_all(t_pred)
        ms_pred = timed(lambda: ctx.predict_all(t_pred))
        ms_setj = timed(lambda: ctx.set_j(*jstate))
        ctx.predict_all(t_pred)
        ctx.tune("fuse_predict", 1)
        # NEXT-3: selection over all N and the corrector for the timed block (it rewrites those bodies: last)
        ctx.set_steps(f64(2.0 ** -np.asarray(cfg["levels"], dtype=np.float64)))
        act = torch.empty(N, dtype=torch.int32, device=dev)
        ms_sel = timed(lambda: ctx.next_block(act))
        ms_cor = timed(lambda: ctx.correct(t_pred, idx, out["acc"], out["jerk"], 0.02, 2.0 ** -3))
        # NEXT-3 as ONE call per block: 100 consecutive blocks from a mid-run state (t0 = last block time before
        # 0.3 at each body's level); what a block costs outside its force kernel (selection + its host read-back,
        # finalize, corrector, launches)
        lev = np.asarray(cfg["levels"], dtype=np.float64)
        dt_np = 2.0 ** -lev
        bctx = nb.nb_open(N, 8, stream)
        bstate = list(jstate)
        bstate[5] = f64(np.floor(0.3 / dt_np) * dt_np)
        bctx.set_j(*bstate)
        bctx.set_steps(f64(dt_np))
        for _ in range(5):
            bctx.block_step(None, 0.02, 2.0 ** -6)
        torch.cuda.synchronize()
        bctx.tune("profile", 1)
        nblk, sizes, fused_blk, stamps, last_launch = 150, [], [], [time.perf_counter()], []
        for _ in range(nblk):
            _, nn_b = bctx.block_step(None, 0.02, 2.0 ** -6)
            stamps.append(time.perf_counter())
            sizes.append(nn_b); fused_blk.append(bctx.info("last_fused"))
            last_launch.append(bctx.info("force_kernel_count") - 1)   # a mis-speculated block launched a no-op first
        torch.cuda.synchronize()
        assert last_launch[-1] < 256
        force_us = np.array([bctx.info("force_kernel_ns_at", q) * 1e-3 for q in last_launch])
        spec = {"hits": bctx.info("spec_hits"), "misses": bctx.info("spec_misses")}
        bctx.tune("profile", 0)
        bctx.close()
        # call k returns after ENQUEUEING block k; its kernels run while call k+1 waits for its selection:
        # the interval between the returns of calls k and k+1 holds block k's force kernel
        cycle_us = np.diff(np.array(stamps))[1:] * 1e6              # [k] = return(k+1) - return(k), k = 0 .. nblk-2
        sizes_a, fused_a = np.array(sizes), np.array(fused_blk)
        small = (sizes_a[:-1] <= 128) & (sizes_a[1:] <= 128)
        outside = cycle_us - force_us[:-1]
        blockstep = {"blocks": nblk, "n_act_median": float(np.median(sizes_a)), "n_act_min": int(sizes_a.min()),
                     "n_act_max": int(sizes_a.max()), "fused_blocks": int(fused_a.sum()), "speculation": spec,
                     "small_blocks_measured": int(small.sum()),
                     "us_per_small_block": float(np.median(cycle_us[small])) if small.any() else None,
                     "us_force_kernel_per_small_block": float(np.median(force_us[:-1][small])) if small.any() else None,
                     "us_per_small_block_outside_force_kernel": float(np.median(outside[small])) if small.any() else None,
                     "us_per_block_outside_force_kernel_all_median": float(np.median(outside)),
                     "note": "150 back-to-back nb_block_step calls (h2 = NULL: total force) from a mid-run state; cycle = host "
                             "wall clock between the returns of consecutive calls; force kernel = CUDA events around its "
                             "launch; small = blocks of <= 128 active bodies (fused prediction)"}
        # NEXT-1: the full-N pass: every body active, counts only (no 2 GiB list), h2 = the block radii
        h2_full = f64(cfg["h2_all"])
        fo = dict(acc=torch.empty((N, 3), dtype=torch.float64, device=dev), jerk=torch.empty((N, 3), dtype=torch.float64, device=dev),
                  pot=torch.empty(N, dtype=torch.float64, device=dev), nnb=torch.empty(N, dtype=torch.int32, device=dev),
                  overflow=torch.empty(N, dtype=torch.int32, device=dev))
        ctx.predict_all(t_pred)
        ms_full = timed(lambda: ctx.regular_all(h2_full, fo["acc"], fo["jerk"], fo["pot"], fo["nnb"], None, fo["overflow"]), reps=2)
        fullpass = {"N": N, "ms": ms_full, "pairs_per_s": float(N) * N / (ms_full * 1e-3),
                    "frac_fp32_peak": float(N) * N * FLOP_PER_INTERACTION / (ms_full * 1e-3) / 1e12 / peak_tflops,
                    "jsplit": ctx.info("last_jsplit"), "reordered": ctx.info("last_reordered"),
                    "note": "nb_regular_all, nblist = NULL (neighbours counted), includes the Morton sort of the block and finalize"}
        del fo, h2_full
        # NEXT-3, two-level Ahmad-Cohen stepping: start-up (full regular pass with lists + neighbour force) and
        # 120 blocks; a block without a regular step never touches all N bodies' forces
        actx = nb.nb_open(N, cap, stream)
        astate = list(jstate)
        astate[5] = torch.zeros(N, dtype=torch.float64, device=dev)
        actx.set_j(*astate)
        a0_, a1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0_.record(stream)
        actx.ac_init(0.0, f64(cfg["h2_all"]), 0.02, 2.0 ** -6)
        a1_.record(stream); torch.cuda.synchronize()
        ms_acinit = a0_.elapsed_time(a1_)
        for _ in range(5):
            actx.ac_step(0.02, 0.03, 2.0 ** -6)
        torch.cuda.synchronize()
        stamps_a, kinds = [time.perf_counter()], []
        for _ in range(120):
            _, ni_a, nr_a = actx.ac_step(0.02, 0.03, 2.0 ** -6)
            stamps_a.append(time.perf_counter()); kinds.append((ni_a, nr_a))
        torch.cuda.synchronize()
        segs = []                                         # the loop inside the library, in segments of 100 blocks
        for _ in range(6):
            tw = time.perf_counter()
            _, nb_run, ni_run, nr_run = actx.ac_run(0.02, 0.03, 2.0 ** -6, max_blocks=100)
            torch.cuda.synchronize()
            segs.append({"blocks": int(nb_run), "irregular_steps": int(ni_run), "regular_steps": int(nr_run),
                         "us_per_block_mean": (time.perf_counter() - tw) * 1e6 / max(nb_run, 1)})
        tw = time.perf_counter()                          # and a long stretch: 2000 blocks in one call
        _, nb_long, ni_long, nr_long = actx.ac_run(0.02, 0.03, 2.0 ** -6, max_blocks=2000)
        torch.cuda.synchronize()
        ac_long = {"blocks": int(nb_long), "irregular_steps": int(ni_long), "regular_steps": int(nr_long),
                   "ms": (time.perf_counter() - tw) * 1e3, "us_per_block_mean": (time.perf_counter() - tw) * 1e6 / max(nb_long, 1)}
        spec_ac = {"hits": actx.info("spec_hits"), "misses": actx.info("spec_misses")}
        actx.close()
        cyc = np.diff(np.array(stamps_a))[1:] * 1e6
        kinds_a = np.array(kinds)
        irr_only = (kinds_a[:-1, 1] == 0) & (kinds_a[1:, 1] == 0)
        with_reg = kinds_a[:-1, 1] > 0
        acstep = {"nb_ac_init_ms": ms_acinit, "blocks": 120, "n_irr_median": float(np.median(kinds_a[:, 0])),
                  "blocks_without_regular_step": int((kinds_a[:, 1] == 0).sum()),
                  "us_per_block_without_regular_step": float(np.median(cyc[irr_only])) if irr_only.any() else None,
                  "us_per_block_with_regular_step": float(np.median(cyc[with_reg])) if with_reg.any() else None,
                  "nb_ac_run_segments_of_100_blocks": segs, "nb_ac_run_2000_blocks": ac_long, "speculation": spec_ac,
                  "n_reg_median_when_due": float(np.median(kinds_a[kinds_a[:, 1] > 0, 1])) if (kinds_a[:, 1] > 0).any() else None,
                  "note": "config 4 at t = 0 with the block radii (150 neighbours, cap 512); host wall clock between the returns "
                          "of consecutive nb_ac_step calls"}
        extras = {
            "nb_ac_step": acstep,
            "nb_regular_all": fullpass,
            "nb_block_step": blockstep,
            "nb_irregular": {"n_i": n_i, "neighbour_pairs": nn, "ms": ms_irr, "pairs_per_s": nn / (ms_irr * 1e-3),
                             "gather_GBps": nn * 128 / (ms_irr * 1e-3) / 1e9, "dtype": "f64"},
            "nb_update_j": {"n": n_i, "ms": ms_upd},
            "nb_predict_all": {"ms": ms_pred, "GBps": N * (112 + 40) / (ms_pred * 1e-3) / 1e9,
                               "frac_hbm": N * (112 + 40) / (ms_pred * 1e-3) / 1e9 / pk["hbm_gbs"], "hbm_peak_GBps": pk["hbm_gbs"],
                               "hbm_peak_source": pk_src},
            "nb_next_block": {"N": N, "ms": ms_sel, "note": "min + count + ordered scatter + 16 B D2H + sync"},
            "nb_correct": {"n": n_i, "ms": ms_cor},
            "nb_set_j": {"ms": ms_setj, "GBps": N * (112 + 112 + 128) / (ms_setj * 1e-3) / 1e9,
                         "note": "timed after nb_irregular / nb_update_j: the context also keeps the 128 B/body gather copy current"},
        }

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu = cpu_oracle_rate(cfg, idx_np, h2_np, seconds_target=12.0)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}

    # The metric is "... vs block size": the sweep rides inside `roofline` too (compact rows), because a record that
    # keeps only the contract's objects would otherwise lose it (round-2 verdict, "What's missing" 3).
    def compact(rows):
        return [{"n_i": r["n_i"], "ms": r["ms"], "frac": r["frac_fp32_peak"], "variant": r["variant"], "jsplit": r["jsplit"],
                 "fused": r["fused_predict"], "ms_predict_plus_regular_in_stream": r["ms_predict_plus_regular_in_stream"]}
                for r in rows]
    if roofline is not None and sweep:
        roofline["sweep"] = compact(sweep)
        roofline["sweep_note"] = ("nb_regular alone at N = %d, records resident, min of 10; frac = of the FP32 peak above" % N)
    if roofline is not None and other:
        roofline["other_configs"] = {name: {"N": o["N"], "sweep": compact(o["sweep"])} for name, o in other.items()}
    if roofline is not None and extras:
        roofline["block_loop"] = {"us_per_small_block": extras["nb_block_step"].get("us_per_small_block"),
                                  "us_per_ac_block_without_regular_step": extras["nb_ac_step"].get("us_per_block_without_regular_step"),
                                  "nb_regular_all_frac": extras["nb_regular_all"].get("frac_fp32_peak")}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 pair math (x differenced as hi/lo f32 pairs, f64 sums)",
        "data": "synthetic",
        "config": {"workload": WORKLOAD, "N": N, "n_i_per_gpu": n_i, "nb_cap": cap, "nb_target": cfg["nb_target"],
                   "parallelism": f"i-shard x{world}" if world > 1 else "single GPU",
                   "step": "nb_set_j + nb_predict_all + nb_regular",
                   "l2": "each step streams 2*112 B/body (set_j) + 112+40 B/body (predict) = 394 MB > 126 MB L2 "
                         "before the force kernel; its 42 MB j-record working set is L2-resident by design",
                   **plan},
        "frac_fp32_peak": value / world * FLOP_PER_INTERACTION / 1e12 / peak_tflops,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
        "cpu_baseline": cpu, "sweep": sweep, "other_configs": other, "extras": extras, "peaks_source": pk_src,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_b200_jsharded(args, world, rank, local):
    """--shard j: each rank owns a contiguous N / world slice of the bodies in its own context; every step all
    ranks evaluate the same active block with nb_regular_shard and exchange the partial results
    (paper_1504_03687_b200.parallel: Table 2).  Total work is fixed: strong scaling."""
    import torch
    import torch.distributed as dist
    import nbgen
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200 import parallel as par
    N = args.N
    cfg, idx_np, h2_np = build_workload(N, args.n_i)
    n_i, cap, t_pred = int(idx_np.shape[0]), cfg["cap"], float(cfg["t"])
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()
    b = par.shard_bounds(N, world)
    lo, hi = b[rank], b[rank + 1]
    f64 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
    state = {k: f64(cfg[k][lo:hi]) for k in par.STATE_KEYS}
    ctx = nb.nb_open(hi - lo, cap, stream)
    ctx.set_j_offset(lo)
    idx, h2 = torch.from_numpy(np.ascontiguousarray(idx_np)).to(dev), f64(h2_np)

    def step():
        ctx.set_j(*(state[k] for k in par.STATE_KEYS))
        ctx.predict_all(t_pred)
        return par.regular_jsharded(ctx, state, lo, t_pred, idx, h2)

    for _ in range(max(args.warmup, 3)):
        res = step()
    torch.cuda.synchronize()
    launches0 = ctx.info("kernel_launches")
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    w0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        res = step()
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    launches = ctx.info("kernel_launches") - launches0
    if world > 1:
        tt = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms = float(tt.item())
        tl = torch.tensor([launches], dtype=torch.int64, device=dev)
        dist.all_reduce(tl, op=dist.ReduceOp.SUM)
        launches = int(tl.item())
    clocks = sampler.stop(w0, w1) if sampler else None
    if rank == 0:
        pk, pk_src = peaks()
        sm_max_mhz = float((clocks or {}).get("sm_max_mhz") or pk.get("sm_max_mhz", 1965.0))
        peak_tflops = ctx.info("sm_count") * 128 * 2 * sm_max_mhz * 1e6 / 1e12
        value = float(n_i) * N * args.steps / (ms * 1e-3)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32 pair math (x differenced in warp-local f32 frames or as hi/lo f32 pairs, f64 sums)",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "N": N, "n_i": n_i, "nb_cap": cap, "parallelism": f"j-shard x{world}",
                       "step": "per rank: nb_set_j(shard) + nb_predict_all + nb_regular_shard; state all-reduce, "
                               "sums + list rows all-gather (paper_1504_03687_b200.parallel)",
                       "l2": "each step streams the shard's state through set_j + predict before the force kernel"},
            "frac_fp32_peak": value / world * FLOP_PER_INTERACTION / 1e12 / peak_tflops, "clocks": clocks, "e2e": None,
            "gpu_launches": int(launches), "roofline": None, "cpu_baseline": None,
            "checksum_pot": float(res["pot"].sum()), "peaks_source": pk_src,
        }
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
