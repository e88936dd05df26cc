#!/usr/bin/env python
"""bench.py -- submatrix sign-function hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one seeded synthetic workload:
sm_build_pattern -> sm_gather -> sm_sign_ns -> sm_scatter -> D = 1/2 (I - R), Tr D
(all rows of SURVEY.md section 8(a)), inputs resident in HBM.  Default workload: BASELINE.json
configs[2] (3,000 molecules x 23 orbitals, cutoff 5 A, bf16 in / fp32 accumulate, 20 fixed
Newton-Schulz iterations) -- one of the two configurations the metric's roofline target is quoted on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl reference]

Prints ONE JSON line (rank 0).  `value` = effective TFLOP/s = 4 * sum_i m_i^3 * k / step time over
all ranks (true m_i, no padding, no symmetry discount).  See DESIGN.md section 7 for every field.
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

from workloads.generator import CONFIGS, make_config  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (mean of its PHASE 1 / PHASE 2 launches),
# from the committed `ncu --set full` captures under profiles/ (r1c_ncu_full_k_umma_gemm_cfg{2,4}.md, r1b_ncu_full_k_dmma_gemm_cfg1.md).
NCU_TRAFFIC_BYTES = {(2, "bf16"): 3.47e9, (4, "bf16"): 28.8e9, (1, "f64"): 0.72e9}

METRIC = "submatrix_sign_effective_tflops"
UNIT = "TFLOP/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--run", type=int, default=0, help="index into the config's precision runs")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scale", default=None, help="none|gershgorin|power|global (default: global for 16-bit, gershgorin otherwise)")
    ap.add_argument("--h-dtype", default=None, choices=["f64", "f32"], help="storage type of the H values (default: f32 for 16-bit runs, f64 otherwise)")
    ap.add_argument("--chunk-elems", type=int, default=0, help="cap on the packed elements per chunk of sm_density (0: one chunk if it fits)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload_stats(wl):
    cnt_dim = np.array([wl.blk_size[wl.col_idx[wl.row_ptr[i]:wl.row_ptr[i + 1]]].sum()
                        for i in range(wl.n_blk)], dtype=np.float64)
    return cnt_dim, float((cnt_dim ** 3).sum())


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm=d.get("hbm_gbs", 6650.0), burst=d.get("bf16_tflops", 1590.0),
                    sustained=d.get("bf16_tflops_sustained", 1400.0), src="measured")
    return dict(hbm=6650.0, burst=1590.0, sustained=1400.0, src="fallback")


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(wl, cfg_run, n_cols_sample, seed, n_threads):
    """Times the oracle, as it stands, on a seeded sample of block columns.  Returns
    (seconds, flop-equivalent = 4 sum m^3 k over the sample, columns)."""
    from oracle import oracle as orc
    from workloads.generator import sample_columns
    cols = sample_columns(wl, n_cols_sample, seed)
    m = np.array([wl.blk_size[wl.col_idx[wl.row_ptr[i]:wl.row_ptr[i + 1]]].sum() for i in cols], dtype=np.float64)
    k = cfg_run["max_iter"] if cfg_run["tol"] <= 0 else 15   # convergence runs: ~15 updates
    t0 = time.perf_counter()
    orc.density_columns(wl, cols=cols, n_threads=n_threads)
    dt = time.perf_counter() - t0
    return dt, 4.0 * float((m ** 3).sum()) * k, cols


def oracle_sample_size(cfg_index, cores):
    # ~10-30 s of CPU work: per-submatrix cost of the Jacobi oracle ~ 2.2e-8 * m^3 s (measured here)
    per = {0: 0.003, 1: 0.25, 2: 4.0, 3: 0.25, 4: 600.0}[cfg_index]      # cfg2: 32 columns took 7 s on 16 cores
    return max(1, min(int(20.0 * cores / per), {0: 32, 1: 1000, 2: 3000, 3: 10000, 4: 2000}[cfg_index])) \
        if per < 100 else max(1, min(cores, 8))


def run_reference(args, cfg, cfg_run):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_config(args.config)
    cores = os.cpu_count() or 1
    n_sample = oracle_sample_size(args.config, cores)
    for w in range(args.warmup):
        oracle_sample(wl, cfg_run, max(1, n_sample // 8), 7000 + w, cores)
    total_t, total_f, total_cols = 0.0, 0.0, 0
    for s in range(args.steps):
        dt, fl, cols = oracle_sample(wl, cfg_run, n_sample, 9000 + s, cores)
        total_t += dt; total_f += fl; total_cols += len(cols)
    val = total_f / total_t / 1e12
    sample = f"{n_sample} seeded block columns of {cfg['name']} per step (of {wl.n_blk})"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": cfg["name"], "x_dtype": cfg_run["x_dtype"],
                                        "sample": sample},
        "block_columns_per_s": total_cols / total_t,
        "cpu_baseline": {"value": val, "unit": UNIT + " (equivalent: 4*sum m^3*k_gpu / t_oracle)",
                         "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, cfg, cfg_run):
    import torch
    import torch.distributed as dist
    import paper_2205_14741_b200.binding as sm   # raises if the CUDA library is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    x_dtype = cfg_run["x_dtype"]
    is16 = x_dtype in ("bf16", "f16")
    pad = 64 if is16 else 16
    # 16-bit, fixed iteration counts: SM_SCALE_GLOBAL (one interlacing bound from power steps on the block-sparse
    # matrix; same error class as the per-submatrix power scale, no second gather -- DESIGN.md A10)
    scale_mode = args.scale or ("global" if is16 else "gershgorin")
    max_iter, tol = cfg_run["max_iter"], cfg_run["tol"]

    # Weak scaling: every rank owns an independent replica of the workload (independent problems,
    # PAPER.md:106 "large-scale parallel evaluation"); no data-path collective.
    from paper_2205_14741_b200 import dist_util
    wl = make_config(args.config, seed=dist_util.rank_seed(cfg["seed"], rank))
    dims, sum_m3 = workload_stats(wl)
    # H storage (SURVEY 8(d) G5 / reading A16): the fp64 master copy for the fp64 / fp32 runs, an fp32 copy for the
    # 16-bit runs (cast once on the host when the workload is made; X0 is rounded from fp32 arithmetic either way)
    h_dtype = args.h_dtype or ("f32" if is16 else "f64")
    hb = {"f64": 8, "f32": 4}[h_dtype]
    A = sm.Bcsr(wl, val_dtype=h_dtype)
    P = sm.sm_build_pattern(A, pad)
    eb = {"f64": 8, "f32": 4, "bf16": 2, "f16": 2}[x_dtype]
    free_b, _ = torch.cuda.mem_get_info()
    budget = int(0.25 * free_b / eb)
    max_chunk = P.packed_elems if P.packed_elems <= budget else max(budget, P.max_dim_pad ** 2)
    if args.chunk_elems > 0:
        max_chunk = max(min(max_chunk, args.chunk_elems), P.max_dim_pad ** 2)
    plan = sm.DensityPlan(A, P, x_dtype, max_chunk_elems=max_chunk)

    def step():
        # a1 runs every step; its size query (a validation pass plus a read-back that synchronises the stream) is
        # per geometry and was done once above
        Pn = sm.sm_build_pattern(A, pad, sizes=P.sizes)
        sm.sm_density(A, Pn, plan, mu=0.0, scale_mode=scale_mode, max_iter=max_iter, tol=tol, symmetrise=True)
        return Pn

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sm.launch_count()
    sm.profile_enable(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    ms_total = ev0.elapsed_time(ev1)
    gemm_ms, gemm_launches = sm.profile_read()
    sm.profile_enable(False)
    launches = sm.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    iters_mean = float(plan.iters.double().mean().item())
    k_eff = plan.iters.double().cpu().numpy()
    order = P.order.cpu().numpy()
    flops_step = 4.0 * float(((dims[order] ** 3) * k_eff).sum())    # per-column updates actually applied
    ms_total_max, flops_all = dist_util.aggregate(ms_total, flops_step, torch.device("cuda", local))
    ms_per_step = ms_total_max / args.steps
    value = flops_all / (ms_per_step * 1e-3) / 1e12

    # ---- stage breakdown (one extra untimed-for-headline pass, CUDA events per stage)
    stages = {}
    if rank == 0:
        def timed(fn):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); a.record(); out = fn(); b.record(); torch.cuda.synchronize()
            return out, a.elapsed_time(b)
        Pn, stages["pattern_ms"] = timed(lambda: sm.sm_build_pattern(A, pad))
        free_now, _ = torch.cuda.mem_get_info()
        if max_chunk >= P.packed_elems and 3.3 * P.packed_elems * eb < free_now:   # X + Y + X' of a separate pass
            cols, col_off, n = sm.sm_plan_columns(Pn, Pn.order)
            X, sc = sm.sm_gather(A, Pn, cols, col_off, n, 0.0, scale_mode, x_dtype)     # untimed: first-use allocations
            (X, sc), stages["gather_ms"] = timed(lambda: sm.sm_gather(A, Pn, cols, col_off, n, 0.0, scale_mode, x_dtype, X=X))
            ws = torch.empty(sm.sm_sign_ws_bytes(Pn, n, Pn.packed_elems, x_dtype), dtype=torch.uint8, device="cuda")
            _, stages["sign_ms"] = timed(lambda: sm.sm_sign_ns(Pn, cols, col_off, n, Pn.packed_elems, x_dtype, X,
                                                               max_iter, tol, ws=ws))
            R, stages["scatter_ms"] = timed(lambda: sm.sm_scatter(A, Pn, cols, col_off, n, x_dtype, X, "f64",
                                                                 R=plan.D, symmetrise=True))
            _, stages["density_ms"] = timed(lambda: sm.sm_density_from_sign(A, Pn, R))
            stages["sign_tflops"] = flops_step / (stages["sign_ms"] * 1e-3) / 1e12
            e_x = eb
            stages["gather_gbs"] = (Pn.packed_elems * e_x + A.n_vals * hb + Pn.gmap_len * 4) / (stages["gather_ms"] * 1e-3) / 1e9
            del X, ws

    # ---- end to end through the public call with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        h_vals = torch.from_numpy(np.ascontiguousarray(wl.vals, dtype=np.float32 if h_dtype == "f32" else np.float64)).pin_memory()
        h_D = torch.empty(A.n_vals, dtype=torch.float64).pin_memory()
        h_tr = torch.empty(1, dtype=torch.float64).pin_memory()
        h_idx = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in
                 (wl.blk_size.astype(np.int32), wl.row_ptr.astype(np.int32), wl.col_idx.astype(np.int32),
                  wl.val_ptr.astype(np.int64))]
        d_idx = [A.blk_size, A.row_ptr, A.col_idx, A.val_ptr]

        # Software pipeline over steps: step k's input copies (copy-in stream) and result copies (copy-out stream)
        # overlap the compute of the neighbouring steps; every step still moves its own inputs from pinned host
        # memory and its own D and Tr D back, all inside the timed region.  Two sets of device inputs and outputs
        # (the large workspace is shared: compute is serial on the main stream).
        import copy
        A_b = [A, sm.Bcsr(wl, val_dtype=h_dtype)]
        plan_b = [plan, copy.copy(plan)]
        plan_b[1].D = torch.zeros_like(plan.D); plan_b[1].trace = torch.zeros_like(plan.trace)
        plan_b[1].iters = torch.zeros_like(plan.iters); plan_b[1].residual = torch.zeros_like(plan.residual)
        plan_b[1].scale = torch.zeros_like(plan.scale)
        h_Db = [h_D, torch.empty_like(h_D).pin_memory()]
        h_trb = [h_tr, torch.empty_like(h_tr).pin_memory()]
        s_main = torch.cuda.current_stream()
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        ev_in = [torch.cuda.Event() for _ in range(2)]
        ev_done = [torch.cuda.Event() for _ in range(2)]
        ev_out = [torch.cuda.Event() for _ in range(2)]

        def e2e_step(k):
            b_ = k & 1
            Ab, pb = A_b[b_], plan_b[b_]
            with torch.cuda.stream(s_in):
                s_in.wait_event(ev_done[b_])            # the step that last read these inputs has finished
                for h, d in zip(h_idx, (Ab.blk_size, Ab.row_ptr, Ab.col_idx, Ab.val_ptr)):
                    d.copy_(h, non_blocking=True)
                Ab.vals.copy_(h_vals, non_blocking=True)
                ev_in[b_].record(s_in)
            s_main.wait_event(ev_in[b_])
            s_main.wait_event(ev_out[b_])               # this buffer's previous result has left the device
            Pn = sm.sm_build_pattern(Ab, pad, sizes=P.sizes)
            sm.sm_density(Ab, Pn, pb, mu=0.0, scale_mode=scale_mode, max_iter=max_iter, tol=tol, symmetrise=True)
            ev_done[b_].record(s_main)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_done[b_])
                h_Db[b_].copy_(pb.D, non_blocking=True)
                h_trb[b_].copy_(pb.trace, non_blocking=True)
                ev_out[b_].record(s_out)
        e2e_step(0); e2e_step(1)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for k in range(args.steps):
            e2e_step(k)
        s_main.wait_stream(s_out)
        b.record()
        torch.cuda.synchronize()
        e2e_ms = dist_util.aggregate(a.elapsed_time(b), 0.0, torch.device("cuda", local))[0] / args.steps
        h2d = int(h_vals.numel() * hb + sum(x.numel() * x.element_size() for x in h_idx))
        d2h = int(h_D.numel() * 8 + 8)
        e2e = {"value": flops_all / (e2e_ms * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "pipelining": "copy-in / compute / copy-out on three streams, double-buffered inputs and outputs"}

    if rank != 0:
        if world > 1:
            dist.barrier(); dist.destroy_process_group()
        return

    peaks = load_peaks()
    if is16:
        # dominant kernel: k_umma_gemm.  Algorithmic FLOPs per launch = 2 sum m^3 (one m x m x m product per
        # submatrix); launches inside the timed region = 2 * k * steps.  With SM_UMMA_FUSED=1 one launch of
        # k_umma_fused runs all 2 k products, so the per-launch figure is the total over the timed launches.
        long_region = ms_total_max > 4000.0
        peak = peaks["sustained"] if long_region else peaks["burst"]
        flops_per_launch = flops_step * args.steps / max(gemm_launches, 1)
        avg_ms = gemm_ms / max(gemm_launches, 1)
        achieved = flops_per_launch / (avg_ms * 1e-3) / 1e12
        fused = os.environ.get("SM_UMMA_FUSED", "0")[:1] == "1"
        roofline = {"bound": "tensor", "kernel": "k_umma_fused" if fused else "k_umma_gemm", "achieved": achieved, "peak": peak,
                    "unit": "TFLOP/s", "frac": achieved / peak,
                    "traffic": None if fused else NCU_TRAFFIC_BYTES.get((args.config, x_dtype)),
                    "peak_source": f"{peaks['src']} bf16 {'sustained' if long_region else 'burst'}",
                    "launches_timed": gemm_launches, "avg_launch_ms": avg_ms,
                    "algorithmic_flops_per_launch": flops_per_launch}
    else:
        # fp64: DMMA tensor path (k_dmma_gemm); fp32: FFMA (k_simt_gemm).  Peak derived:
        # 148 SMs x 64 (fp64) / 128 (fp32) FMA per clock x 2 x 1.965 GHz.  Algorithmic FLOPs per launch = the
        # products actually run: 2 sum_i m_i^3 k_i / (launches / 2 per step) -- convergence mode drops columns.
        peak = 37.2 if x_dtype == "f64" else 74.4
        avg_ms = gemm_ms / max(gemm_launches, 1)
        flops_per_launch = flops_step * args.steps / max(gemm_launches, 1)
        achieved = flops_per_launch / (avg_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "k_dmma_gemm" if x_dtype == "f64" else "k_simt_gemm",
                    "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                    "traffic": NCU_TRAFFIC_BYTES.get((args.config, x_dtype)),
                    "peak_source": "derived: 148 SMs x FMA lanes x 2 x 1.965 GHz",
                    "launches_timed": gemm_launches, "avg_launch_ms": avg_ms,
                    "algorithmic_flops_per_launch": flops_per_launch,
                    "note": "fp64 kernel computes lower-triangle tiles only (symmetric iterates): achieved counts the "
                            "full 2 m^3 per product and may exceed the derived peak" if x_dtype == "f64" else None}

    cpu = None
    if not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_sample = oracle_sample_size(args.config, cores)
        dt, fl_eq, cols = oracle_sample(make_config(args.config), cfg_run, n_sample, 9000, cores)
        cpu = {"value": fl_eq / dt / 1e12, "unit": UNIT + " (equivalent: 4*sum m^3*k_gpu / t_oracle)",
               "cores": cores, "kind": "oracle", "block_columns_per_s": len(cols) / dt, "seconds": dt,
               "sample": f"{len(cols)} seeded block columns of {cfg['name']} (of {wl.n_blk}), fp64 Jacobi"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": x_dtype, "data": "synthetic",
        "config": {"workload": cfg["name"], "n_mol": cfg["n_mol"], "orbitals": cfg["b"], "cutoff_A": cfg["cutoff"],
                   "x_dtype": x_dtype, "max_iter": max_iter, "tol": tol, "scale_mode": scale_mode, "h_dtype": h_dtype, "pad_to": pad,
                   "l2": "inputs_exceed_l2" if P.packed_elems * eb > 200e6 else "inputs_fit_l2",
                   "chunks": int(-(-P.packed_elems // max_chunk))},
        "block_columns_per_s": world * wl.n_blk / (ms_per_step * 1e-3),
        "iters_mean": iters_mean, "trace": float(plan.trace.item()),
        "residual_max": float(plan.residual.max().item()),
        "stages": stages, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
        "gpu_launches": int(launches), "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier(); dist.destroy_process_group()


def main():
    args = parse_args()
    cfg = CONFIGS[args.config]
    cfg_run = cfg["runs"][args.run]
    if args.impl == "reference":
        run_reference(args, cfg, cfg_run)
    else:
        run_ours(args, cfg, cfg_run)


if __name__ == "__main__":
    main()
