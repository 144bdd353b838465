#!/usr/bin/env python
"""bench.py -- the headline measurement of the GP prediction pipeline (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl b200|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

One "step" is one pass of the whole hot path over one batch of
synthetic NFIR-shaped input: assemble K, tiled Cholesky, both
triangular solves, predictive mean, full predictive covariance.  Every phase is bracketed by CUDA
events on the launching stream; `value` is the Cholesky rate n^3/3 / t_cholesky summed over all
ranks (replicas only: each GPU factors its own problem, no data-path collective, DESIGN.md
"Multi-GPU").  Rank 0 prints ONE JSON line.

`--impl reference` times the CPU oracle (oracle/, the only reference this tier has) on a bounded
sample of the same workload on the box's host cores.

Extras (not part of the default line): `--sweep` runs the config-2 tile-size x scheduler-width
sweep (analogue of the paper's Fig. 3) and `--cusolver-ref` times cuSOLVER potrf
once through torch.linalg.cholesky as a reported reference; both print JSON lines
of their own.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FP64 tiled Cholesky GFLOP/s and full-cov prediction time at n=32768; % FP64 peak"

# DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the dominant kernel
# (exec_kernel<128>, the Cholesky DAG) comes from the ncu --set full captures summarised under
# profiles/: profiles/ncu_traffic.json records, per (n, tile), the bytes, the capture it came from, the
# commit and the fingerprint of the work-item schedule it was taken with.  bench.py reports the
# figure only while the library still builds the same schedule, else null.
NCU_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")

ORACLE_SAMPLE = (4096, 512)             # (n, m) of the sampled oracle pipeline pass (configs 3-4) and of --impl reference
ORACLE_CHOLESKY_SIZES = (4096, 8192)    # measured unblocked-Cholesky passes the n^3 extrapolation starts from (configs 3-4)
ORACLE_CHOLESKY_SIZES_LONG = (4096, 8192, 16384)   # with --cpu-baseline-long (minutes of CPU)
E2E_UNIT = "GFLOP/s"                    # identical in both arms, so that the driver can form e2e_ratio


def _parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (default 3: the headline)")
    ap.add_argument("--tile", type=int, default=0, help="override the config's tile size")
    ap.add_argument("--width", type=int, default=0, help="scheduler width (persistent CTAs), 0 = one per SM")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-baseline-long", action="store_true",
                    help="configs 3-4: also time the oracle's Cholesky at n=16384; config 2: also the 1-thread full pass")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "block-cyclic", "shard-predict"],
                    help="N > 1 only. replicas (default): N independent problems, weak scaling, no data-path collective. "
                         "block-cyclic: ONE factorisation, tile columns distributed over the ranks, panels broadcast (NCCL), strong "
                         "scaling (SURVEY 8(f) row 2). shard-predict: replicated factor, prediction sharded by test-point tile rows "
                         "with one all-gather of V^T, strong scaling (SURVEY 8(e)). The last two are unmeasured on hardware.")
    ap.add_argument("--fused-bcast", action="store_true",
                    help="--mode block-cyclic: the panel step writes the panel into the other ranks' memory (gp_mixed_panel_bcast over CUDA IPC "
                         "peer mappings) instead of an NCCL broadcast after it; unverified on multi-GPU hardware")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--cusolver-ref", action="store_true")
    ap.add_argument("--ozaki-probe", action="store_true", help="bounds of the emulated contraction (measurement support, one JSON line)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, f"/tmp/gp_b200_clocks_{os.getpid()}.csv"

    def start(self):
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.f.close()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        with open(self.path) as f:
            for line in f:
                p = [x.strip() for x in line.split(",")]
                if len(p) < 7:
                    continue
                try:
                    sm.append(float(p[0])); smax.append(float(p[1])); power.append(float(p[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, p[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        try:
            os.remove(self.path)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # samples under load = upper half (the sampler also sees the idle edges of the region)
        load = sorted(sm)[len(sm) // 2:]
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


def reduce_max_over_ranks(values, device="cpu"):
    """Element-wise MAX of per-rank timings over the default process group (a no-op at world size 1)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def replica_seeds(config_index: int, rank: int):
    """Every replica factors its own problem of the same shape (replicas only)."""
    return 1000 + config_index + 10 * rank, 2000 + config_index + 10 * rank


def aggregate_cholesky_gflops(n: int, world: int, cholesky_ms_max_over_ranks: float) -> float:
    """Whole-job rate: the n^3/3 flop of every replica over the slowest rank's time."""
    return world * (n ** 3 / 3.0) / (cholesky_ms_max_over_ranks * 1e-3) / 1e9


def _dist_env():
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    return rank, local, world


def _config(args):
    from paper_2602_19683_b200 import nfir
    cfg = nfir.CONFIGS[args.config]
    tile = args.tile or cfg.tile
    return cfg, tile


def _config_dict(cfg, tile, width, world):
    M = cfg.n // tile
    return {"workload": f"c{cfg.index}: n={cfg.n} m={cfg.m} D={cfg.D} tile={tile} ({M}x{M} tiles) FP64, NFIR-shaped synthetic",
            "n": cfg.n, "m": cfg.m, "D": cfg.D, "tile": tile, "sched_width": width or "auto (one CTA per SM)",
            "lengthscale": cfg.lengthscale, "vertical": cfg.vertical, "noise": cfg.noise,
            "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)",
            "l2": "inputs larger than L2 (K tiles %.2f GB re-assembled every step)" % (M * (M + 1) / 2 * tile * tile * 8 / 1e9)}


# ------------------------------------------------------------------------------------------------
def oracle_run(n, m, D, cfg, seed_shift=0, cholesky_only=False):
    """One oracle pass (a1-a12, or a1-a6 with cholesky_only) on an (n, m) sample of the workload's
    generator; returns per-phase seconds."""
    import oracle
    from paper_2602_19683_b200 import nfir
    X, y = nfir.nfir_features(1000 + cfg.index + seed_shift, n, D)
    Xs, _ = nfir.nfir_features(2000 + cfg.index + seed_shift, m, D, with_targets=False)
    h = oracle.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    t0 = time.perf_counter()
    K = oracle.assemble(X, X, h, True)
    t1 = time.perf_counter()
    L = oracle.cholesky(K)
    t2 = time.perf_counter()
    if cholesky_only:
        return {"assemble_s": t1 - t0, "cholesky_s": t2 - t1, "predict_s": None, "total_s": t2 - t0}
    beta = oracle.forward_subst(L, y)
    alpha = oracle.backward_subst(L, beta)
    fitted = oracle.Prediction(K=None, L=L, beta=beta, alpha=alpha)
    oracle.predict(X, y, Xs, h, full_cov=True, fitted=fitted)
    t3 = time.perf_counter()
    return {"assemble_s": t1 - t0, "cholesky_s": t2 - t1, "predict_s": t3 - t2, "total_s": t3 - t0}


def cpu_baseline(cfg, long_run=False):
    """The oracle as it stands on the box's host cores.
    Configs 0-2: the FULL oracle on the same config, all threads, and a 1-thread time beside it (config 2:
    the 1-thread pass only with --cpu-baseline-long: it is minutes).  Configs 3-4: the full oracle would run
    for many minutes, so the Cholesky is MEASURED at n = 4096 and 8192 (16384 too with --cpu-baseline-long)
    and the figure for the config's own n is the n^3 scaling of the largest measured pass, under the key
    `extrapolated` (optimistic for the CPU: the unblocked oracle is memory-bound and slows down with n);
    the prediction phase is measured on an (n=4096, m=512) sample."""
    import oracle
    threads = oracle.num_threads()
    flop = lambda n: n ** 3 / 3.0
    if cfg.index <= 2:
        r = oracle_run(cfg.n, cfg.m, cfg.D, cfg)
        out = {"value": flop(cfg.n) / r["cholesky_s"] / 1e9, "unit": "GFLOP/s", "cores": threads, "kind": "oracle",
               "sample": f"the full oracle on the same config (n={cfg.n}, m={cfg.m}, D={cfg.D}), one pass, {threads} threads",
               "cholesky_ms": r["cholesky_s"] * 1e3, "predict_full_cov_ms": r["predict_s"] * 1e3, "pipeline_ms": r["total_s"] * 1e3}
        if cfg.index < 2 or long_run:
            oracle.set_num_threads(1)
            try:
                r1 = oracle_run(cfg.n, cfg.m, cfg.D, cfg)
            finally:
                oracle.set_num_threads(threads)
            out["one_thread"] = {"value": flop(cfg.n) / r1["cholesky_s"] / 1e9, "cholesky_ms": r1["cholesky_s"] * 1e3,
                                 "predict_full_cov_ms": r1["predict_s"] * 1e3, "pipeline_ms": r1["total_s"] * 1e3}
        else:
            out["one_thread"] = None      # run with --cpu-baseline-long
        return out
    sizes = ORACLE_CHOLESKY_SIZES_LONG if long_run else ORACLE_CHOLESKY_SIZES
    measured = []
    for n in sizes:
        r = oracle_run(n, 32, cfg.D, cfg, cholesky_only=True)
        measured.append({"n": n, "cholesky_s": r["cholesky_s"], "gflops": flop(n) / r["cholesky_s"] / 1e9})
    ns, ms = ORACLE_SAMPLE
    rp = oracle_run(ns, ms, cfg.D, cfg)
    last = measured[-1]
    ext_s = last["cholesky_s"] * (cfg.n / last["n"]) ** 3
    return {"value": last["gflops"], "unit": "GFLOP/s", "cores": threads, "kind": "oracle",
            "sample": f"unblocked oracle Cholesky MEASURED at n={', '.join(str(x['n']) for x in measured)} (D={cfg.D}, same generator, "
                      f"{threads} threads); value = the rate of the largest measured pass; the figure for n={cfg.n} is extrapolated",
            "measured": measured,
            "extrapolated": {"n": cfg.n, "cholesky_s": ext_s, "gflops": flop(cfg.n) / ext_s / 1e9,
                             "how": f"t(n) = t({last['n']}) * (n/{last['n']})^3: flop scaling only, optimistic for the CPU "
                                    "(the unblocked oracle is memory-bound and its rate falls as n grows)"},
            "pipeline_sample": {"n": ns, "m": ms, "cholesky_ms": rp["cholesky_s"] * 1e3, "predict_full_cov_ms": rp["predict_s"] * 1e3,
                                "pipeline_ms": rp["total_s"] * 1e3}}


def reference_sample(cfg):
    """(n, m) one step of --impl reference runs: the config itself where the oracle finishes it in seconds
    (configs 0-1), otherwise a bounded sample of the same generator."""
    if cfg.index <= 1:
        return cfg.n, cfg.m, False
    return min(ORACLE_SAMPLE[0], cfg.n), min(ORACLE_SAMPLE[1], cfg.m), True


def run_reference(args):
    rank, _, world = _dist_env()
    if rank != 0:
        return 0
    import oracle
    cfg, tile = _config(args)
    n, m, sampled = reference_sample(cfg)
    for _ in range(args.warmup):
        oracle_run(n, m, cfg.D, cfg)
    chol, total, pred = 0.0, 0.0, 0.0
    for s in range(args.steps):
        r = oracle_run(n, m, cfg.D, cfg)
        chol += r["cholesky_s"]; total += r["total_s"]; pred += r["predict_s"]
    value = args.steps * (n ** 3 / 3.0) / chol / 1e9
    sample = (f"each step = one oracle pass (a1-a12) on an n={n}, m={m}, D={cfg.D} SAMPLE of the same generator" if sampled
              else f"each step = one oracle pass (a1-a12) on the config itself (n={n}, m={m}, D={cfg.D})")
    config = _config_dict(cfg, tile, args.width, world)
    if sampled:     # say what was actually run: the oracle cannot finish this config within the driver's time
        config["workload"] = (f"SAMPLE n={n} m={m} D={cfg.D} of " + config["workload"] +
                              " -- the unblocked CPU oracle runs a bounded sample, not the config")
        config["sample_n"], config["sample_m"] = n, m
    e2e_value = args.steps * (n ** 3 / 3.0) / total / 1e9     # same definition as the b200 arm: n^3/3 over the whole pipeline time
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
            "predict_full_cov_ms": pred / args.steps * 1e3, "gpu_launches": 0,
            "cpu_baseline": {"value": value, "unit": "GFLOP/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            # the oracle has no device: its end-to-end figure is the line's own value and unit (0 bytes copied); the rate over
            # its whole pipeline time (the b200 arm's e2e definition) is given beside it
            "e2e": {"value": value, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                    "pipeline_value": e2e_value,
                    "pipeline_definition": "n^3/3 of the problem actually run over its whole pipeline time (a1-a12)"}}
    print(json.dumps(line), flush=True)
    return 0


def ncu_traffic(gp, n, tile):
    """DRAM bytes of one Cholesky launch from profiles/ncu_traffic.json, or None when there is no capture for
    this workload or the library no longer builds the schedule the capture was taken with."""
    try:
        table = json.load(open(NCU_TRAFFIC_FILE))
    except (OSError, ValueError):
        return None, "no profiles/ncu_traffic.json"
    rec = table.get(f"n={n},tile={tile}")
    if rec is None:
        return None, "no ncu capture for this workload"
    fp = "%016x" % gp.gp_schedule_fingerprint(n, 0, tile, 148)
    if rec.get("schedule_fingerprint") != fp:
        return None, f"stale: captured with schedule {rec.get('schedule_fingerprint')} at {rec.get('commit')}, this build makes {fp}"
    return float(rec["dram_bytes"]), f"{rec.get('source')} (commit {rec.get('commit')})"


# ------------------------------------------------------------------------------------------------
def measure_fp64_peak(gp, torch):
    """DMMA / DFMA register-resident microbenchmarks: burst (best of 10 short launches) and
    sustained (back to back for ~2 s), in TFLOP/s."""
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    out = {}
    for mode, name in ((0, "dmma"), (1, "dfma")):
        iters = 20000 if mode == 0 else 40000
        for _ in range(3):
            flops = gp.gp_fp64_peak_launch(mode, iters, sink)
        torch.cuda.synchronize()
        best = 0.0
        for _ in range(10):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); gp.gp_fp64_peak_launch(mode, iters, sink); b.record(); torch.cuda.synchronize()
            best = max(best, flops / (a.elapsed_time(b) * 1e-3) / 1e12)
        out[name + "_burst_tflops"] = best
        if mode == 0:
            one = flops / (best * 1e12)
            reps = max(4, int(2.0 / one))
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                gp.gp_fp64_peak_launch(mode, iters, sink)
            b.record(); torch.cuda.synchronize()
            out["dmma_sustained_tflops"] = reps * flops / (a.elapsed_time(b) * 1e-3) / 1e12
    # the contraction path alone (TMA stream + DMMA loop + epilogue + signalling, no DAG): K = 1024 items
    K, reps = 1024, 100
    buf = (torch.rand(gp.gp_contraction_bench_bytes(K, reps) // 8 + 1, dtype=torch.float64, device="cuda") * 1e-3).view(torch.uint8)
    for _ in range(2):
        flops = gp.gp_contraction_bench_launch(K, reps, buf)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); flops = gp.gp_contraction_bench_launch(K, reps, buf); b.record(); torch.cuda.synchronize()
    out["contraction_k1024_tflops"] = flops / (a.elapsed_time(b) * 1e-3) / 1e12
    del buf
    # the same contraction emulated on the int8 tensor cores (7 planes of 8-bit digits, 28 int8 GEMMs)
    ma = nb = 8192; kk = 4096
    A = torch.rand(ma, kk, dtype=torch.float64, device="cuda") - 0.5
    Ap = gp.gp_ozaki_slice(A, 2.0)
    C = torch.zeros(ma, nb, dtype=torch.float64, device="cuda")
    best = 0.0
    for r in range(4):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); gp.gp_ozaki_contract(Ap, Ap, 2.0, 2.0, C); b.record(); torch.cuda.synchronize()
        if r > 0:
            best = max(best, 2.0 * ma * nb * kk / (a.elapsed_time(b) * 1e-3) / 1e12)
    out["ozaki_int8_contraction_fp64_equivalent_tflops"] = best
    S = gp.gp_ozaki_planes()
    out["ozaki_int8_pops"] = best * (S * (S + 1) // 2) / 1e3
    del A, Ap, C
    out["int8_mma_peak_pops"] = measure_int8_peak(gp, torch, 128)["pops"]
    return out


def measure_int8_peak(gp, torch, n_cols):
    """Bare tcgen05.mma kind::i8 issue loop (128 x n_cols x 32) on every SM: burst rate in int8 POPS (best of 5 launches of
    ~1 ms) and CTA 0's cycles per MMA."""
    cyc = torch.zeros(1, dtype=torch.int64, device="cuda")
    iters = 2000
    ops = gp.gp_int8_mma_peak_launch(n_cols, iters, cyc)
    torch.cuda.synchronize()
    best = 0.0
    for _ in range(5):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); gp.gp_int8_mma_peak_launch(n_cols, iters, cyc); b.record(); torch.cuda.synchronize()
        best = max(best, ops / (a.elapsed_time(b) * 1e-3) / 1e15)
    return {"pops": best, "cycles_per_mma": float(cyc.item()) / (16.0 * iters)}


def run_ozaki_probe(args):
    """Where the emulated contraction's time goes (profiles/r02_ozaki_bounds.md): the tensor core's int8 rate by a bare issue
    loop for three MMA widths, and the 128 x 128 two-pass kernel with its parts switched off, on random and on constant
    operands (the board's power limit makes the rate depend on how many bits toggle)."""
    import torch
    from paper_2602_19683_b200 import binding as gp
    gp.load()
    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    sampler.start()
    out = {"what": "bench.py --ozaki-probe", "mma_issue_loop": {}, "kernel": []}
    for n_cols in (64, 128, 256):
        out["mma_issue_loop"][f"128x{n_cols}x32"] = measure_int8_peak(gp, torch, n_cols)
    S = gp.gp_ozaki_planes()
    pairs = S * (S + 1) // 2
    m = 8192
    for kind in ("random", "constant"):
        for k in (1024, 4096, 16384):
            A = (torch.rand(m, k, dtype=torch.float64, device="cuda") - 0.5) * 1.8 if kind == "random" else torch.full((m, k), 0.3, dtype=torch.float64, device="cuda")
            Ap = gp.gp_ozaki_slice(A, 2.0)
            del A
            C = torch.zeros(m, m, dtype=torch.float64, device="cuda")
            row = {"operands": kind, "m": m, "n": m, "k": k}
            for probe, name in ((0, "full"), (1, "no_tma_loads"), (2, "loads_only"), (4, "no_reductions_into_c")):
                gp.gp_ozaki_probe_launch(probe, Ap, Ap, C); torch.cuda.synchronize()
                best = 1e30
                for _ in range(3):
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(); gp.gp_ozaki_probe_launch(probe, Ap, Ap, C); b.record(); torch.cuda.synchronize()
                    best = min(best, a.elapsed_time(b))
                row[name] = {"ms": best, "tflops_fp64_equivalent": 2.0 * m * m * k / (best * 1e-3) / 1e12, "int8_pops": 2.0 * m * m * k * pairs / (best * 1e-3) / 1e15}
                if probe in (1, 4) or (probe == 0 and False):
                    pass
                if probe != 0:
                    t = gp.gp_ozaki_probe_stamps()
                    mm0, mm1 = (k // 128) * 4 * sum(1 for p in range(S) for q in range(S) if p + q <= S // 2 - 1), 0
                    mm1 = (k // 128) * 4 * pairs - mm0
                    row[name]["stamps_cycles"] = {"pass0_issue": t[1] - t[0], "pass1_issue": t[3] - t[2], "pass0_epilogue": t[5] - t[4], "pass1_epilogue": t[7] - t[6],
                                                  "pass0_cycles_per_mma": (t[1] - t[0]) / mm0, "pass1_cycles_per_mma": (t[3] - t[2]) / mm1}
            out["kernel"].append(row)
            del Ap, C
    out["clocks"] = sampler.stop()
    print(json.dumps(out), flush=True)
    return 0


LAUNCHES_PER_STEP = {"assemble": 1, "cholesky": 1, "solve": 3, "mean": 1, "full_cov": 5}   # kernels of libgp_b200.so


def run_distributed(args):
    """--mode block-cyclic / shard-predict: one problem on N GPUs (strong scaling), paper_2602_19683_b200/multi_gpu.py."""
    import torch
    import torch.distributed as dist
    rank, local, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2602_19683_b200 import binding as gp, multi_gpu as mg, nfir
    gp.load()
    cfg, tile = _config(args)
    n, m, D = cfg.n, cfg.m, cfg.D
    h = gp.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    X, y, Xs = nfir.make_inputs(cfg)                       # the SAME problem on every rank
    dX, dY, dXs = (torch.from_numpy(a).cuda() for a in (X, y, Xs))
    pipe = gp.GpPipeline(n, 0, D, tile, h, sched_width=args.width)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    times = []
    if args.mode == "block-cyclic":
        peers, keep = (), None
        if world > 1 and args.fused_bcast:      # panels stored straight into the other ranks' copies (NVLink peer memory)
            peers, keep = mg.exchange_peer_pointers(pipe.KL)
        st = mg.MixedCholeskyRank(n, tile, pipe.KL, pipe.info, rank, world, args.width, peers)
        for it in range(args.warmup + args.steps):
            pipe.assemble(dX)
            st.reset()
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            if world > 1:
                st.run()
            else:
                mg.run_lockstep([st])
            b.record()
            barrier()
            if it >= args.warmup:
                times.append(a.elapsed_time(b))
        what = ("Cholesky, tile columns block-cyclic over the ranks, FP64 panels " +
                ("stored into every rank's copy by the panel step itself (fused broadcast over peer memory)" if peers else "broadcast with NCCL") +
                ", int8-emulated trailing updates")
    else:
        pipe.assemble(dX); pipe.cholesky(); pipe.solve(dY)   # replicated factor (not timed)
        sp = mg.ShardedPredictor(n, m, D, tile, h, rank, world, args.width)
        for it in range(args.warmup + args.steps):
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            sp.solve_local(pipe.KL, dX, dXs, pipe.alpha)
            if world > 1:
                sp.all_gather()
            sp.covariance_rows(dXs)
            b.record()
            barrier()
            if it >= args.warmup:
                times.append(a.elapsed_time(b))
        what = "full-covariance prediction given L, sharded by test-point tile rows, one all-gather of V^T"
    ms = reduce_max_over_ranks([sum(times) / len(times)], device="cuda")[0]
    if rank == 0:
        flop = n ** 3 / 3.0 if args.mode == "block-cyclic" else float(n) * n * m + 2.0 * n * m * m
        cfgd = _config_dict(cfg, tile, args.width, world)
        cfgd["parallelism"] = f"{args.mode} over {world} GPU(s): {what}"
        print(json.dumps({"metric": METRIC, "value": flop / (ms * 1e-3) / 1e9, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f64 panels + int8-emulated updates" if args.mode == "block-cyclic" else "f64", "data": "synthetic",
                          "config": cfgd, "mode": args.mode, "info": int(pipe.info.item()),
                          "note": "multi-GPU path verified by one-GPU lock-step emulation and gloo tests; unmeasured on multi-GPU hardware"}),
              flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_b200(args):
    import torch
    rank, local, world = _dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl b200 needs a CUDA device: there is no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2602_19683_b200 import binding as gp, nfir
    gp.load()
    cfg, tile = _config(args)
    n, m, D = cfg.n, cfg.m, cfg.D
    h = gp.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    # every replica gets its own seeded problem of the same shape
    seed_train, seed_test = replica_seeds(cfg.index, rank)
    X, y = nfir.nfir_features(seed_train, n, D)
    Xs, _ = nfir.nfir_features(seed_test, m, D, with_targets=False)
    hX, hY, hXs = (torch.from_numpy(a).pin_memory() for a in (X, y, Xs))
    dX, dY, dXs = hX.cuda(), hY.cuda(), hXs.cuda()
    # step a6, host half: build + upload the static schedules once, outside every timed region (the first
    # compute call for a shape would otherwise do it, blocking the host; include/gp_b200.h)
    schedule_build_ms = gp.gp_prepare(n, m, tile, gp.GP_PREPARE_CHOLESKY | gp.GP_PREPARE_FULL_COV | gp.GP_PREPARE_VARIANCE)
    pipe = gp.GpPipeline(n, m, D, tile, h, sched_width=args.width)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    names = ("assemble", "cholesky", "solve", "mean", "full_cov")

    def step(ev=None):
        def mark(i):
            if ev is not None:
                ev[i].record()
        mark(0); pipe.assemble(dX)
        mark(1); pipe.cholesky()
        mark(2); pipe.solve(dY)
        mark(3); gp.gp_predict_mean(dX, pipe.alpha, dXs, h, pipe.mean)
        mark(4); gp.gp_predict_full_cov(pipe.KL, dX, dXs, h, tile, args.width, pipe.Sigma, pipe.work)
        mark(5)

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    events = [[torch.cuda.Event(enable_timing=True) for _ in range(6)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    for s in range(args.steps):
        step(events[s])
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    info = int(pipe.info.item())
    # cheap parity guard on the LAST timed step's outputs (full parity is tests/test_gpu_full_size.py): alpha must solve
    # K alpha = y.  K alpha = sum_j k(x_i, x_j) alpha_j + noise alpha_i comes from the library's own fused kernel-matrix
    # product (gp_predict_mean with the training points as test points), so the check runs no library linear algebra;
    # a wrong block anywhere in L, beta or alpha shows up here at O(1).  Outside every timed region.
    Ka = torch.empty(n, dtype=torch.float64, device="cuda")
    gp.gp_predict_mean(dX, pipe.alpha, dX, h, Ka)
    Ka += cfg.noise * pipe.alpha
    resid = float((Ka - dY).norm() / dY.norm())
    del Ka
    phase = {nm: sum(events[s][i].elapsed_time(events[s][i + 1]) for s in range(args.steps)) for i, nm in enumerate(names)}
    total_ms = sum(events[s][0].elapsed_time(events[s][5]) for s in range(args.steps))
    per_step_chol = [events[s][1].elapsed_time(events[s][2]) for s in range(args.steps)]

    phase_full_cov_ms = phase["full_cov"] / args.steps
    # SURVEY.md 8(f) rows 1 and 4, outside the step (reported next to it): variance-only prediction given L and
    # the log marginal likelihood, median of 3 after one warm-up
    var = torch.empty(m, dtype=torch.float64, device="cuda")
    lml = torch.empty(1, dtype=torch.float64, device="cuda")
    tv, tl = [], []
    for r in range(4):
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record(); gp.gp_predict_variance(pipe.KL, dX, dXs, h, tile, args.width, var, pipe.work)
        e[1].record(); gp.gp_log_marginal_likelihood(pipe.KL, n, tile, dY, pipe.alpha, lml)
        e[2].record(); torch.cuda.synchronize()
        if r > 0:
            tv.append(e[0].elapsed_time(e[1])); tl.append(e[1].elapsed_time(e[2]))
    next_rows = {"predict_variance_ms": statistics.median(tv), "log_marginal_likelihood_ms": statistics.median(tl),
                 "log_marginal_likelihood": float(lml.item()), "variance_min_max": [float(var.min().item()), float(var.max().item())]}
    del var, lml
    # the same factorisation with its trailing updates emulated on the int8 tensor cores
    # (gp_cholesky_tiled_mixed, opt-in), reported beside the FP64 DMMA path; median of 3 after one warm-up, and the
    # distance of its factor from the FP64 path's (lower triangle, via gp_tiles_to_dense)
    if tile % 128 == 0 and n // tile <= 60 and n <= 65536:
        L64 = pipe.dense_L()
        mwork = torch.empty(gp.gp_mixed_workspace_bytes(n, tile), dtype=torch.uint8, device="cuda")
        tmx = []
        for r in range(4):
            pipe.assemble(dX)
            e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            e[0].record(); gp.gp_cholesky_tiled_mixed(pipe.KL, n, tile, args.width, pipe.info, mwork); e[1].record(); torch.cuda.synchronize()
            if r > 0:
                tmx.append(e[0].elapsed_time(e[1]))
        Lmx = pipe.dense_L()
        mixed_ms = statistics.median(tmx)
        next_rows["cholesky_mixed_int8_emulated"] = {
            "ms": mixed_ms, "gflops_fp64_equivalent": n ** 3 / 3.0 / (mixed_ms * 1e-3) / 1e9, "info": int(pipe.info.item()),
            "rel_diff_to_fp64_factor": float((Lmx - L64).norm() / L64.norm()),
            "what": "FP64 POTRF/TRSM tile tasks on the executor + SYRK/GEMM tile tasks as split-operand int8 products (7 planes of 8-bit digits) "
                    "(tcgen05.mma kind::i8, TMEM accumulators); not the headline: dtype of `value` stays f64"}
        del L64, Lmx, mwork
        pipe.assemble(dX); pipe.cholesky(); pipe.solve(dY)       # leave the FP64 factor behind for what follows
        if m <= 65536:
            # ... and the full-covariance prediction on the same emulated contraction (given L), beside the FP64 one
            gp.gp_predict_full_cov(pipe.KL, dX, dXs, h, tile, args.width, pipe.Sigma, pipe.work)
            S64 = pipe.Sigma.clone()
            pwork = torch.empty(gp.gp_mixed_predict_workspace_bytes(n, m, tile), dtype=torch.uint8, device="cuda")
            tpx = []
            for r in range(4):
                e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
                e[0].record(); gp.gp_predict_full_cov_mixed(pipe.KL, dX, dXs, h, tile, args.width, pipe.Sigma, pwork); e[1].record()
                torch.cuda.synchronize()
                if r > 0:
                    tpx.append(e[0].elapsed_time(e[1]))
            next_rows["full_cov_mixed_int8_emulated"] = {
                "ms": statistics.median(tpx), "fp64_path_ms": phase_full_cov_ms,
                "rel_diff_to_fp64_sigma": float((pipe.Sigma - S64).norm() / S64.norm()),
                "what": "gp_predict_full_cov_mixed: V^T solve and W = V^T V as split-operand int8 products, TRSM with the diagonal tiles in FP64"}
            varm = torch.empty(m, dtype=torch.float64, device="cuda")
            tvx = []
            for r in range(3):
                e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
                e[0].record(); gp.gp_predict_variance_mixed(pipe.KL, dX, dXs, h, tile, args.width, varm, pwork); e[1].record()
                torch.cuda.synchronize()
                if r > 0:
                    tvx.append(e[0].elapsed_time(e[1]))
            next_rows["predict_variance_mixed_int8_emulated"] = {
                "ms": statistics.median(tvx), "fp64_path_ms": next_rows["predict_variance_ms"],
                "max_abs_diff_to_diag_of_fp64_sigma": float((varm - torch.diagonal(S64)).abs().max())}
            del S64, pwork, varm
    torch.cuda.empty_cache()

    # end to end through the host-buffer C-ABI call: H2D of X, y, X^ and D2H of mean, Sigma inside
    ws = torch.empty(gp.gp_pipeline_workspace_bytes(n, m, D, tile), dtype=torch.uint8, device="cuda")
    hMean = torch.empty(m, dtype=torch.float64).pin_memory()
    hSigma = torch.empty(m, m, dtype=torch.float64).pin_memory()
    del pipe
    for _ in range(min(args.warmup, 2)):
        gp.gp_pipeline_host(hX, hY, hXs, h, tile, args.width, hMean, hSigma, None, ws)
    barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        info_e2e = gp.gp_pipeline_host(hX, hY, hXs, h, tile, args.width, hMean, hSigma, None, ws)
    b.record()
    barrier()
    e2e_ms = a.elapsed_time(b)
    del ws
    # the same host-to-host call with the int8-emulated factorisation and covariance (reported beside the headline)
    if "cholesky_mixed_int8_emulated" in next_rows and m <= 65536:
        torch.cuda.empty_cache()
        wsm = torch.empty(gp.gp_pipeline_mixed_workspace_bytes(n, m, D, tile), dtype=torch.uint8, device="cuda")
        gp.gp_pipeline_host(hX, hY, hXs, h, tile, args.width, hMean, hSigma, None, wsm, mixed=True)
        reps = max(1, min(args.steps, 3))
        a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a2.record()
        for _ in range(reps):
            info_m = gp.gp_pipeline_host(hX, hY, hXs, h, tile, args.width, hMean, hSigma, None, wsm, mixed=True)
        b2.record(); torch.cuda.synchronize()
        next_rows["pipeline_host_mixed_int8_emulated"] = {"ms": a2.elapsed_time(b2) / reps, "fp64_path_ms": e2e_ms / args.steps, "info": info_m,
                                                          "call": "gp_pipeline_host_mixed (pinned host buffers; a1-a12 + copies)"}
        del wsm

    t = reduce_max_over_ranks([phase[nm] for nm in names] + [total_ms, e2e_ms], device="cuda")
    phase = {nm: t[i] / args.steps for i, nm in enumerate(names)}
    total_ms, e2e_ms = t[5] / args.steps, t[6] / args.steps

    if rank == 0:
        flop = n ** 3 / 3.0
        chol_gflops = aggregate_cholesky_gflops(n, world, phase["cholesky"])
        peaks = measure_fp64_peak(gp, torch)
        peak = peaks["dmma_sustained_tflops"]
        achieved = flop / (phase["cholesky"] * 1e-3) / 1e12
        traffic, traffic_source = ncu_traffic(gp, n, tile)
        try:
            mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            mp = {}
        line = {
            "metric": METRIC, "value": chol_gflops, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": _config_dict(cfg, tile, args.width, world),
            "cholesky_ms": phase["cholesky"], "cholesky_ms_per_step": per_step_chol,
            # PAPER.md:163 protocol: mean with a 95 % confidence interval (normal approximation), and the median
            "cholesky_ms_stats": {"mean": statistics.mean(per_step_chol), "median": statistics.median(per_step_chol),
                                  "ci95": (1.96 * statistics.stdev(per_step_chol) / len(per_step_chol) ** 0.5) if len(per_step_chol) > 1 else None,
                                  "runs": len(per_step_chol)},
            "predict_full_cov_ms": phase["solve"] + phase["mean"] + phase["full_cov"],
            "phases_ms": phase, "info": info, "residual_K_alpha_minus_y_last_step": resid,
            "schedule_build_ms": schedule_build_ms,
            "pct_fp64_peak": 100.0 * achieved / peak,
            "e2e": {"value": world * flop / (e2e_ms * 1e-3) / 1e9, "unit": E2E_UNIT,
                    "definition": "n^3/3 over the whole host-to-host pipeline time (a1-a12 + copies)", "ms": e2e_ms, "h2d_bytes_per_step": (n * D + n + m * D) * 8, "d2h_bytes_per_step": (m + m * m) * 8 + 4,
                    "info": info_e2e, "call": "gp_pipeline_host (pinned host buffers)"},
            "gpu_launches": sum(LAUNCHES_PER_STEP.values()) * args.steps,
            "roofline": {"bound": "tensor", "kernel": "exec_kernel<128> (tiled Cholesky DAG: POTRF/TRSM/SYRK/GEMM; TMA-fed FP64 DMMA)",
                         "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
                         "compulsory_bytes": (n // tile) * (n // tile + 1) * tile * tile * 8,   # read K once + write L once
                         "peak_source": "gp_fp64_peak_launch DMMA.8x8x4 register-resident microbenchmark, measured live, "
                                        "sustained ~2 s loop (kernel is timed inside a long step)",
                         "peak_burst": peaks["dmma_burst_tflops"], "dfma_burst": peaks["dfma_burst_tflops"],
                         "frac_of_burst": achieved / peaks["dmma_burst_tflops"],
                         "contraction_alone_tflops": peaks["contraction_k1024_tflops"],
                         "emulated_contraction_tflops_fp64_equivalent": peaks["ozaki_int8_contraction_fp64_equivalent_tflops"],
                         "emulated_contraction_int8_pops": peaks["ozaki_int8_pops"],
                         "int8_mma_peak_pops": peaks["int8_mma_peak_pops"],
                         "emulated_contraction_frac_of_int8_peak": peaks["ozaki_int8_pops"] / peaks["int8_mma_peak_pops"],
                         "int8_peak_source": "gp_int8_mma_peak_launch: bare tcgen05.mma kind::i8 128x128x32 issue loop on every SM, burst, live "
                                             "(MEASURED_PEAKS.json has no int8 figure; its bf16 burst x the nominal ratio 2 is given beside it)",
                         "int8_peak_from_bf16_pops": (2.0 * mp["bf16_tflops"] / 1e3) if mp.get("bf16_tflops") else None,
                         "full_cov_exec_tflops": (n * n * m + n * m * m) / (phase["full_cov"] * 1e-3) / 1e12,
                         "hbm_gbs_measured": mp.get("hbm_gbs"),
                         "assemble_gbs": (n // tile) * (n // tile + 1) / 2 * tile * tile * 8 / (phase["assemble"] * 1e-3) / 1e9,
                         "solve_gbs": 2 * (n // tile) * (n // tile + 1) / 2 * tile * tile * 8 / (phase["solve"] * 1e-3) / 1e9},
            "clocks": clocks,
            "next_rows": next_rows,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(cfg, args.cpu_baseline_long)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------
def run_sweep(args):
    """Config 2: tile in {256,512,1024} x scheduler width in {1,2,4,8,16,32,64,148}; Cholesky + full-cov
    (the analogue of the paper's stream-count x tile-count sweep, Fig. 3).
    protocol: mean of the repetitions with a 95 % confidence interval (at least 5 repetitions; 10 from width 8)."""
    import torch
    from paper_2602_19683_b200 import binding as gp, nfir
    cfg = nfir.CONFIGS[2]
    n, m, D = cfg.n, cfg.m, cfg.D
    X, y, Xs = nfir.make_inputs(cfg)
    dX, dY, dXs = (torch.from_numpy(a).cuda() for a in (X, y, Xs))
    h = gp.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    rows = []

    def ci95(v):
        return 1.96 * statistics.stdev(v) / len(v) ** 0.5 if len(v) > 1 else None

    for tile in (256, 512, 1024):
        gp.gp_prepare(n, m, tile)
        for width in (1, 2, 4, 8, 16, 32, 64, sms):
            pipe = gp.GpPipeline(n, m, D, tile, h, sched_width=width)
            reps = 5 if width < 8 else 10
            tc, tp = [], []
            for r in range(reps + 1):
                pipe.assemble(dX)
                e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
                e[0].record(); pipe.cholesky(); e[1].record()
                pipe.solve(dY); pipe.predict(dX, dXs, True); e[2].record()
                torch.cuda.synchronize()
                if r > 0:
                    tc.append(e[0].elapsed_time(e[1])); tp.append(e[1].elapsed_time(e[2]))
            rows.append({"tile": tile, "sched_width": width, "reps": reps, "cholesky_ms": statistics.mean(tc), "cholesky_ms_ci95": ci95(tc),
                         "cholesky_gflops": n ** 3 / 3.0 / (statistics.mean(tc) * 1e-3) / 1e9,
                         "predict_full_cov_ms": statistics.mean(tp), "predict_full_cov_ms_ci95": ci95(tp)})
            del pipe
    print(json.dumps({"sweep": "c2 n=8192 m=1024 D=8: tile x scheduler width (PAPER.md:169 analogue)", "rows": rows}), flush=True)
    return 0


def run_cusolver_ref(args):
    """cuSOLVER potrf on the dense matrix, once, as a reported reference only."""
    import torch
    from paper_2602_19683_b200 import binding as gp, nfir
    cfg, tile = _config(args)
    n = cfg.n
    X, _ = nfir.nfir_features(1000 + cfg.index, n, cfg.D)
    dX = torch.from_numpy(X).cuda()
    h = gp.Hyper(cfg.lengthscale, cfg.vertical, cfg.noise)
    K = torch.empty(n * n, dtype=torch.float64, device="cuda")
    gp.gp_assemble_tiles(dX, dX, h, n, gp.GP_GENERAL, K)      # one tile of edge n = the dense matrix
    K = K.view(n, n)
    K.diagonal().add_(cfg.noise)
    torch.linalg.cholesky(K[:1024, :1024].clone())            # library warm-up
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); L = torch.linalg.cholesky(K); b.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    print(json.dumps({"reference_only": "cuSOLVER potrf via torch.linalg.cholesky (out of place, dense)", "n": n, "ms": ms,
                      "gflops": n ** 3 / 3.0 / (ms * 1e-3) / 1e9}), flush=True)
    return 0


def main():
    args = _parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.cusolver_ref:
        return run_cusolver_ref(args)
    if args.ozaki_probe:
        return run_ozaki_probe(args)
    if args.mode != "replicas":
        return run_distributed(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
