#!/usr/bin/env python
"""Benchmark of the R-ChFSI filter hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c1|c2|c3|c4] [--impl ours|reference]

A "step" is one whole rchfsi_filter call (scalars, Lambda recurrence, init, the p-1 fused
operator+recurrence launches, the final combination) on one synthetic block.  Metric
(BASELINE.json): row*vector*degree updates/s = m*N*p / t.  Prints ONE JSON line.
Default workload: BASELINE.json configs[1] (dense generalized, m=4000, N=240, p=25, TF32 apply).
N > 1: the filter is column-separable (no data-path collective), so every rank filters its own
block of N columns against a replica of the operator ("weak" scaling).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "Chebyshev-filter row*vector*degree updates/s"
UNIT = "updates/s"

WORKLOADS = {
    "c1": dict(name="configs[0] dense standard m=1000 N=60 p=20 FP64 + 1e-4 column noise", apply="fp64", store="fp64"),
    "c2": dict(name="configs[1] dense generalized m=4000 N=240 p=25, TF32 apply, FP64 recurrence", apply="tf32", store="fp64"),
    "c3": dict(name="configs[2] 64^3 7-point Laplacian CSR m=262144 N=300 p=30, FP32 SpMM, FP64 recurrence", apply="fp32", store="fp64"),
    "c4": dict(name="configs[3] FE 16^3 cells degree 6 m=912673 N=1200 p=40", apply="tf32", store="fp64"),
    "c5": dict(name="configs[4] FE 24^3 cells degree 6 m=3048625 N=2400 p=50, filter only (FP32 recurrence and residual "
                    "block, FP64 X; BF16 cell-GEMM operands, one BF16 shadow block updated in place)", apply="bf16", store="fp32"),
}


FE_CELLS = None
BLOCK = None


def make_problem(wl):
    """Seeded synthetic problem + filter bounds (recipes: DESIGN.md 'Input recipe')."""
    if wl == "c1":
        p = workloads.config1_dense_standard()
        b = (p["lam_min"], p["lam_T"], p["lam_max"])
    elif wl == "c2":
        p = workloads.config2_dense_generalized()
        # lam(A) in [-2.1, 12.1], lam(B) in [0.79, 1.21], 1/diag(B) ~ 1: 16 bounds lam(B^-1 A) and lam(D^-1 A)
        b = (None, None, 16.0)
    elif wl == "c3":
        p = workloads.config3_sparse_laplacian()
        b = (None, None, p["lam_max"])
    elif wl == "c5":
        p = workloads.config5_fe()
        if FE_CELLS is not None:
            import workloads.fe as wfe
            p = wfe.fe_problem(FE_CELLS, 6, 5, cell_dtype=np.float32)
            p.update(n_wanted=2048, block=2400, degree=50, tol=1e-8, x0_seed=2005)
        b = (None, None, None)
    elif wl == "c4":
        p = workloads.config4_fe()
        if FE_CELLS is not None:
            import workloads.fe as wfe
            p = wfe.fe_problem(FE_CELLS, 6, 4)
            p.update(n_wanted=1000, block=1200, degree=40, tol=1e-8, x0_seed=2004)
        b = (None, None, None)
    else:
        raise SystemExit("unknown workload " + wl)
    if BLOCK is not None:
        p["block"] = BLOCK
        p["n_wanted"] = min(p["n_wanted"], BLOCK)
        p.pop("X0", None)
    return p, b


def fe_lam_max(prob):
    sample = list(range(0, prob["n_cells"], max(1, prob["n_cells"] // 16)))
    return 1.02 * workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"], sample)


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks line):
    NVML (same counters nvidia-smi prints) every 5 ms, falling back to the nvidia-smi query."""

    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
        r = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
        bits = [getattr(n, "nvmlClocksEventReasonHwSlowdown", 0x8), getattr(n, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                getattr(n, "nvmlClocksEventReasonSwThermalSlowdown", 0x20), getattr(n, "nvmlClocksEventReasonSwPowerCap", 0x4)]
        return [sm, self.max_sm] + [bool(r & b) for b in bits]

    def _sample_smi(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                             capture_output=True, text=True, timeout=5).stdout
        f = [x.strip() for x in out.strip().split(",")]
        return [float(f[0]), float(f[1])] + [x == "Active" for x in f[2:6]]

    def run(self):
        while not self.stop_flag:
            try:
                self.rows.append(self._sample_nvml() if self.nvml else self._sample_smi())
            except Exception:
                pass
            time.sleep(0.005 if self.nvml else 0.05)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(r[0] for r in self.rows)
        reasons = [n for k, n in enumerate(self.NAMES) if any(r[2 + k] for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.rows[0][1], "reasons": reasons,
                "samples": len(self.rows), "source": "nvml" if self.nvml else "nvidia-smi"}


def oracle_filter_time(prob, X, ritz, G, p, bounds, max_cols):
    """Time the oracle's filter_rchfsi as it stands on a column subset (columns are independent)."""
    from oracle import chfsi_oracle as orc
    A, B, Dinv = orc.operators_from_workload(prob)
    nc = min(max_cols, X.shape[1])
    reps, dt = 0, 0.0
    while reps < 1 or (dt < 5.0 and reps < 20):     # a bounded sample: at least one filter, ~5-30 s of CPU work
        t0 = time.perf_counter()
        orc.filter_rchfsi(A.apply, Dinv.apply, X[:, :nc].copy(), ritz[:nc], G[:, :nc].copy(), p, *bounds)
        dt += time.perf_counter() - t0
        reps += 1
    return prob["m"] * nc * p * reps / dt, nc, dt


def run_reference(args):
    """--impl reference: the CPU oracle (tier framing: the reference arm is the oracle)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import chfsi_oracle as orc
    prob, b = make_problem(args.workload)
    N, p = prob["block"], prob["degree"]
    A, B, Dinv = orc.operators_from_workload(prob)
    max_cols = {"c1": 60, "c2": 48, "c3": 8, "c4": 2, "c5": 1}[args.workload]
    rng = np.random.default_rng(123)
    X = rng.standard_normal((prob["m"], max_cols))
    ritz = np.sort(rng.uniform(0.0, 1.0, max_cols))
    G = rng.standard_normal((prob["m"], max_cols)) * 1e-3
    lam_max = b[2] if b[2] is not None else fe_lam_max(prob)
    bounds = (b[0] if b[0] is not None else -3.0, b[1] if b[1] is not None else 1.5, lam_max)
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        orc.filter_rchfsi(A.apply, Dinv.apply, X.copy(), ritz, G, p, *bounds)
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * sum(times) / len(times)
    val = prob["m"] * max_cols * p / (ms * 1e-3)
    cores = os.cpu_count()
    sample = "oracle.filter_rchfsi on %d of %d columns (columns are independent), full m and degree" % (max_cols, N)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOADS[args.workload]["name"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_c5(args, prob, As, Bs, dinv, dev, wl, apply_prec, store_prec, world, rank):
    """configs[4] at full size is a memory plan: X FP64 58.5 GB + G FP32 29.3 GB (caller-owned, read in
    place) + R_X, R_Y FP32 58.5 GB + operator copies.  Only the FILTER is timed: the inputs of Alg. 3 are seeded
    synthetic blocks generated on the device (a Rayleigh-Ritz at this size needs the chunked variant),
    and there is no host copy of an 88 GB input set, so no end-to-end number."""
    import torch
    import paper_2503_22652_b200 as P
    m, N, p = prob["m"], prob["block"], prob["degree"]
    gen = torch.Generator(device=dev)
    gen.manual_seed(prob.get("x0_seed", 5) + rank)
    X = torch.empty((m, N), dtype=torch.float64, device=dev)
    for r0 in range(0, m, 65536):                      # row chunks: no second full-size temporary
        X[r0:r0 + 65536].normal_(generator=gen)
    X *= 1.0 / np.sqrt(m)
    G = torch.empty((m, N), dtype=torch.float32, device=dev)
    for r0 in range(0, m, 65536):
        G[r0:r0 + 65536].normal_(generator=gen)
    G *= 1e-3
    ritz = torch.linspace(-9.0, 3.0, N, dtype=torch.float64, device=dev)
    bounds = (-10.0, 3.5, fe_lam_max(prob))
    solver = P.Rchfsi(As, None, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec, g_input_f32=True)
    for _ in range(args.warmup):
        solver.filter(P.METHOD_RCHFSI, X, ritz, G, p, *bounds)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    l0 = solver.launch_count()
    steps = max(1, min(args.steps, 3))
    total_ms, step_ms, step_n = 0.0, 0.0, 0
    for _ in range(steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        solver.filter(P.METHOD_RCHFSI, X, ritz, G, p, *bounds)
        e1.record()
        ms_k, n_k = solver.last_filter_step_ms()
        total_ms += e0.elapsed_time(e1)
        step_ms += ms_k
        step_n += n_k
    launches = solver.launch_count() - l0
    sampler.stop_flag = True
    sampler.join(timeout=2)
    finite = bool(torch.isfinite(X[::4096]).all().item())
    from paper_2503_22652_b200.sharding import reduce_job
    total_ms, updates = reduce_job(total_ms, float(m) * N * p)
    if rank != 0:
        return
    ms_per_step = total_ms / steps
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    sm = step_ms / max(1, step_n)
    byts = 4.0 * m * N * 4 + prob["n_cells"] * prob["n_loc"] ** 2 * (2.0 if apply_prec == "bf16" else 4.0)
    gbs = byts / (sm * 1e-3) / 1e9
    out = {"metric": METRIC, "value": updates / (ms_per_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps,
           "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": apply_prec, "data": "synthetic",
           "config": {"workload": wl["name"], "m": m, "block_N": N, "degree": p, "apply_prec": apply_prec,
                      "store_prec": store_prec, "l2": "inputs (176 GB) far larger than L2",
                      "device_bytes_allocated": int(torch.cuda.memory_allocated()), "output_finite": finite},
           "clocks": sampler.summary(), "gpu_launches": int(launches),
           "e2e": None, "e2e_note": "no host copy of the 88 GB input set exists on this box",
           "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                        "traffic": None, "kernel": "fused FE operator + recurrence step (8 colour launches)",
                        "step_launch_ms": sm, "peak_source": "measured" if peaks else "fallback"}}
    if args.solve:
        # full R-ChFSI solve at this size: memory-light mode of the library (chunked Rayleigh-Ritz, FP32 residual
        # block read in place); the filter-only handle and its 66 GB are released first
        solver.close()
        del G
        torch.cuda.empty_cache()
        for r0 in range(0, m, 65536):
            X[r0:r0 + 65536].normal_(generator=gen)
        so = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec, adaptive_bounds=True)
        t0 = time.perf_counter()
        r = so.solve(P.METHOD_RCHFSI, X, prob["n_wanted"], p, -100.0, 0.0, bounds[2], tol=1e-8, max_iter=args.solve_iters)
        out["solve"] = {"final_residual": float(r["resnorm"][:prob["n_wanted"]].max()), "iters": int(r["iters"]),
                        "converged": bool(r["converged"]), "seconds": time.perf_counter() - t0,
                        "history": [float(x) for x in r["history"]],
                        "evals_first_last_wanted": [float(r["evals"][0]), float(r["evals"][prob["n_wanted"] - 1])],
                        "device_bytes_torch": int(torch.cuda.memory_allocated())}
        so.close()
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--apply-prec", default=None)
    ap.add_argument("--store-prec", default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-solve", action="store_true")
    ap.add_argument("--solve", action="store_true", help="also run rchfsi_solve on c4 (about a minute)")
    ap.add_argument("--solve-method", default="rchfsi", choices=["rchfsi", "chfsi"],
                    help="method of the extra solve (chfsi = Algorithm 2 with the same kernels, the paper's comparator)")
    ap.add_argument("--solve-iters", type=int, default=60)
    ap.add_argument("--fe-cells", type=int, default=None, help="c4 only: cells per direction (profiling a smaller mesh)")
    ap.add_argument("--block", type=int, default=None, help="override the block width N (profiling)")
    args = ap.parse_args()
    global FE_CELLS, BLOCK
    FE_CELLS, BLOCK = args.fe_cells, args.block
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist
    import paper_2503_22652_b200 as P

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    wl = WORKLOADS[args.workload]
    apply_prec = args.apply_prec or wl["apply"]
    store_prec = args.store_prec or wl["store"]
    prob, b = make_problem(args.workload)
    m, N, p, nw = prob["m"], prob["block"], prob["degree"], prob["n_wanted"]
    As, Bs, dinv = P.upload_problem(prob, device=dev)
    noise = dict(noise_eps=prob.get("noise_eps", 0.0), noise_seed=1234) if args.workload == "c1" else {}
    solver = None
    if args.workload != "c5":
        solver = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec, **noise)

    if args.workload == "c5":
        run_c5(args, prob, As, Bs, dinv, dev, wl, apply_prec, store_prec, world, rank)
        return

    # inputs of Alg. 3: B-orthonormal X, Ritz values and G from one Rayleigh-Ritz on a seeded block
    X0 = prob.get("X0")
    if X0 is None:
        X0 = workloads.start_block(m, N, prob.get("x0_seed", 7) + rank)
    X = torch.as_tensor(X0, dtype=torch.float64).to(dev)
    ritz, X, G, res0 = solver.rayleigh_ritz(X)
    rz = ritz.cpu().numpy()
    lam_max = b[2] if b[2] is not None else fe_lam_max(prob)
    lam_min = b[0] if b[0] is not None else float(rz[0]) - 1e-2 * max(1.0, abs(float(rz[0])))
    lam_T = b[1] if b[1] is not None else float(rz[-1]) + 1e-6
    bounds = (lam_min, lam_T, lam_max)
    Xwork = X.clone()

    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def one_step():
        solver.filter(P.METHOD_RCHFSI, Xwork, ritz, G, p, *bounds)

    for _ in range(args.warmup):
        Xwork.copy_(X)
        one_step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = solver.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    step_kernel_ms, step_kernel_n = 0.0, 0
    torch.cuda.synchronize()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                      # L2 flush between timed iterations (outside the event pair)
        ev[k][0].record()
        one_step()
        ev[k][1].record()
        ms_k, n_k = solver.last_filter_step_ms()   # synchronises: CUDA events around the p-1 step launches
        step_kernel_ms += ms_k
        step_kernel_n += n_k
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    launches = solver.launch_count() - l0
    sampler.stop_flag = True
    sampler.join(timeout=2)
    from paper_2503_22652_b200.sharding import reduce_job
    total_ms = sum(a.elapsed_time(bb) for a, bb in ev)
    if world > 1:
        dist.barrier()
    # max over ranks of the device time, sum over ranks of the units (column shards, no data-path collective)
    total_ms, updates = reduce_job(total_ms, float(m) * N * p)
    ms_per_step = total_ms / args.steps
    value = updates / (ms_per_step * 1e-3)

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    Xh = torch.empty((m, N), dtype=torch.float64).pin_memory()
    Gh = G.cpu().pin_memory()
    rh = ritz.cpu().pin_memory()
    Xh.copy_(X)
    e2e_steps = max(1, min(args.steps, 5))
    solver.filter_host(P.METHOD_RCHFSI, Xh, rh, Gh, p, *bounds)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        solver.filter_host(P.METHOD_RCHFSI, Xh, rh, Gh, p, *bounds)
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps
    te = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_ms = float(te.item())
    h2d = Xh.numel() * 8 + Gh.numel() * 8 + rh.numel() * 8
    d2h = Xh.numel() * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel: the per-step operator(+recurrence) launch
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    bf16_peak = peaks.get("bf16_tflops", 1590.0)
    peak_src = "measured" if peaks else "fallback"
    step_ms = step_kernel_ms / max(1, step_kernel_n)
    sb = 8 if store_prec == "fp64" else 4
    if args.workload in ("c1", "c2"):
        flops = 2.0 * m * m * N
        tf = flops / (step_ms * 1e-3) / 1e12
        if apply_prec in ("tf32", "bf16"):
            peak = bf16_peak * (0.5 if apply_prec == "tf32" else 1.0)
            roof = {"bound": "tensor", "achieved": tf, "peak": peak, "unit": "TFLOP/s", "frac": tf / peak,
                    "traffic": None, "kernel": "dense step (operator apply + recurrence epilogue)",
                    "peak_source": peak_src + " bf16 burst x %.1f" % (0.5 if apply_prec == "tf32" else 1.0)}
        else:
            peak = 37.0 if apply_prec == "fp64" else 75.0
            roof = {"bound": "alu", "achieved": tf, "peak": peak, "unit": "TFLOP/s", "frac": tf / peak,
                    "traffic": None, "kernel": "dense SIMT apply + elementwise step", "peak_source": "nominal"}
    else:
        # algorithmic bytes per step: R_Y, R_X, G read once, R_X written once (+ operator bytes)
        if args.workload == "c3":
            opb = prob["vals"].size * 8.0
        else:
            opb = prob["n_cells"] * prob["n_loc"] ** 2 * (2.0 if apply_prec == "bf16" else 4.0)
        byts = 4.0 * m * N * sb + opb
        gbs = byts / (step_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                "traffic": None, "kernel": "fused operator + recurrence step", "peak_source": peak_src}
    roof["step_launch_ms"] = step_ms
    try:   # DRAM bytes per step from the committed ncu --set full capture of this configuration, else null
        tr = json.load(open(os.path.join(ROOT, "profiles", "r01_traffic.json")))
        if FE_CELLS is None and BLOCK is None:
            roof["traffic"] = tr.get("%s:%s:%s" % (args.workload, apply_prec, store_prec))
    except Exception:
        pass

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": {"fp64": "f64", "fp32": "f32", "tf32": "tf32", "bf16": "bf16"}[apply_prec],
           "data": "synthetic",
           "config": {"workload": wl["name"], "m": m, "block_N": N, "degree": p, "apply_prec": apply_prec,
                      "store_prec": store_prec, "l2": "flushed between timed filter calls (512 MiB memset)",
                      "parallelism": "replicas x%d (column shards, no collective)" % world},
           "clocks": sampler.summary(), "gpu_launches": int(launches),
           "e2e": {"value": updates / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                   "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms},
           "roofline": roof, "wall_s_timed_region": t_wall}

    if not args.no_solve and (args.workload in ("c1", "c2", "c3") or args.solve):
        Xs = torch.as_tensor(X0, dtype=torch.float64).to(dev)
        so = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec,
                      adaptive_bounds=(args.workload != "c1"), **noise)
        t0 = time.perf_counter()
        meth = P.METHOD_RCHFSI if args.solve_method == "rchfsi" else P.METHOD_CHFSI
        r = so.solve(meth, Xs, nw, p, lam_min, lam_T, lam_max, tol=1e-8, max_iter=args.solve_iters)
        out["solve"] = {"method": args.solve_method, "final_residual": float(r["resnorm"][:nw].max()),
                        "iters": int(r["iters"]), "converged": bool(r["converged"]),
                        "seconds": time.perf_counter() - t0, "history": [float(x) for x in r["history"]]}
        so.close()

    if not args.no_cpu_baseline:
        Xc, rc, Gc = X.cpu().numpy(), rz, G.cpu().numpy()
        max_cols = {"c1": 60, "c2": 240, "c3": 16, "c4": 2, "c5": 1}[args.workload]
        v, nc, dt = oracle_filter_time(prob, Xc, rc, Gc, p, bounds, max_cols)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                               "sample": "oracle.filter_rchfsi, %d of %d columns, full m and degree, %.1f s" % (nc, N, dt)}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
