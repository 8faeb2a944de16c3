#!/usr/bin/env python
"""Benchmark of the R-ChFSI filter hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c1|c2|c3|c4|c5] [--impl ours|reference]
                    [--apply-prec P] [--store-prec P] [--no-also] [--no-solve] [--no-e2e] [--no-cpu-baseline]

A "step" is one whole rchfsi_filter call (scalars, Lambda recurrence, init, the p-1 fused
operator+recurrence launches, the final combination) on one synthetic block.  Metric
(BASELINE.json): row*vector*degree updates/s = m*N*p / t.  Prints ONE JSON line.

Default workload: BASELINE.json configs[4], the largest single-GPU configuration (FE 24^3 cells, degree 6,
m = 3,048,625, N = 2400, p = 50, BF16 cell-GEMM operands, FP32 recurrence blocks, FP64 X / Rayleigh-Ritz).
The same line carries
  "also"   one sub-record per remaining kernel claim (c2 dense TF32, c3 CSR FP32, c4 FE TF32, c4 FE BF16, and the
           Rayleigh-Ritz rotation on the INT8 tensor pipe against cuBLAS dgemm),
  "solve"  the full configs[4] R-ChFSI solve to 1e-8, certified by the ORACLE's operator on sampled columns,
  "e2e"    the same filter through rchfsi_filter_host (pinned host buffers, column-chunked pipeline),
  "cpu_baseline"  the oracle's filter on a bounded sample on the host cores.
N > 1: the filter is column-separable (no data-path collective), so every rank filters its own
block of N columns against a replica of the operator ("weak" scaling); sub-records are N = 1 only.
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
    "c4": dict(name="configs[3] FE 16^3 cells degree 6 m=912673 N=1200 p=40", apply="tf32", store="fp32"),
    "c5": dict(name="configs[4] FE 24^3 cells degree 6 m=3048625 N=2400 p=50, BF16 cell-GEMM operands, FP32 recurrence "
                    "and residual block, FP64 X / Rayleigh-Ritz", apply="bf16", store="fp32"),
}
# sub-records of the default line: (key, workload, apply, store, max timed steps)
ALSO = [("c2_tf32", "c2", "tf32", "fp64", 20), ("c3_fp32", "c3", "fp32", "fp64", 20),
        ("c4_tf32_fp32store", "c4", "tf32", "fp32", 5), ("c4_bf16_fp32store", "c4", "bf16", "fp32", 5)]
DTYPE = {"fp64": "f64", "fp32": "f32", "tf32": "tf32", "bf16": "bf16"}

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
        if FE_CELLS is not None:
            import workloads.fe as wfe
            p = wfe.fe_problem(FE_CELLS, 6, 5, cell_dtype=np.float32)
            p.update(n_wanted=2048, block=2400, degree=50, tol=1e-8, x0_seed=2005)
        else:
            p = workloads.config5_fe()
        b = (None, None, None)
    elif wl == "c4":
        if FE_CELLS is not None:
            import workloads.fe as wfe
            p = wfe.fe_problem(FE_CELLS, 6, 4)
            p.update(n_wanted=1000, block=1200, degree=40, tol=1e-8, x0_seed=2004)
        else:
            p = workloads.config4_fe()
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

    def finish(self):
        self.stop_flag = True
        self.join(timeout=2)
        return self.summary()

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(r[0] for r in self.rows)
        reasons = [n for k, n in enumerate(self.NAMES) if any(r[2 + k] for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.rows[0][1], "reasons": reasons,
                "samples": len(self.rows), "source": "nvml" if self.nvml else "nvidia-smi"}


# ----------------------------------------------------------------------------------------- CPU side (oracle)
def oracle_sample_time(prob, p_full, bounds, cols, degree, budget_s=8.0, rng_seed=123, inputs=None):
    """Time the oracle's filter_rchfsi as it stands on a bounded sample: `cols` columns (columns are independent)
    and `degree` recurrence steps (the cost per row*vector*degree update does not depend on the degree).  Returns
    (updates/s, description, seconds)."""
    from oracle import chfsi_oracle as orc
    A, B, Dinv = orc.operators_from_workload(prob)
    m = prob["m"]
    if inputs is None:
        rng = np.random.default_rng(rng_seed)
        X = rng.standard_normal((m, cols))
        ritz = np.sort(rng.uniform(bounds[0], bounds[1], cols))
        G = rng.standard_normal((m, cols)) * 1e-3
    else:
        X, ritz, G = (np.ascontiguousarray(a[..., :cols]) for a in inputs)
    reps, dt = 0, 0.0
    while reps < 1 or (dt < budget_s and reps < 20):
        t0 = time.perf_counter()
        orc.filter_rchfsi(A.apply, Dinv.apply, X.copy(), ritz, G, degree, *bounds)
        dt += time.perf_counter() - t0
        reps += 1
    desc = ("oracle.filter_rchfsi, %d of %d columns, degree %d of %d, full m, %d repetition(s), %.1f s"
            % (cols, prob["block"], degree, p_full, reps, dt))
    return m * cols * degree * reps / dt, desc, dt


CPU_SAMPLE = {"c1": (60, 20), "c2": (240, 25), "c3": (16, 30), "c4": (2, 40), "c5": (2, 8)}   # (columns, degree)
REF_SAMPLE = {"c1": (60, 20), "c2": (48, 25), "c3": (8, 30), "c4": (2, 8), "c5": (1, 3)}


def run_reference(args):
    """--impl reference: the CPU oracle (tier framing: the reference arm is the oracle), each step a bounded
    sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import chfsi_oracle as orc
    prob, b = make_problem(args.workload)
    N, p = prob["block"], prob["degree"]
    A, B, Dinv = orc.operators_from_workload(prob)
    cols, deg = REF_SAMPLE[args.workload]
    rng = np.random.default_rng(123)
    X = rng.standard_normal((prob["m"], cols))
    ritz = np.sort(rng.uniform(0.0, 1.0, cols))
    G = rng.standard_normal((prob["m"], cols)) * 1e-3
    lam_max = b[2] if b[2] is not None else fe_lam_max(prob)
    bounds = (b[0] if b[0] is not None else -3.0, b[1] if b[1] is not None else 1.5, lam_max)
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        orc.filter_rchfsi(A.apply, Dinv.apply, X.copy(), ritz, G, deg, *bounds)
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * sum(times) / len(times)
    val = prob["m"] * cols * deg / (ms * 1e-3)
    cores = os.cpu_count()
    sample = ("oracle.filter_rchfsi on %d of %d columns (columns are independent), degree %d of %d, full m"
              % (cols, N, deg, p))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOADS[args.workload]["name"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ----------------------------------------------------------------------------------------- GPU side
def load_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def load_traffic():
    """DRAM bytes per step from the committed ncu --set full captures (profiles/), keyed workload:apply:store."""
    for name in ("r02_traffic.json", "r01_traffic.json"):
        try:
            return json.load(open(os.path.join(ROOT, "profiles", name))), "profiles/%s (ncu --set full, committed)" % name
        except Exception:
            continue
    return {}, None


def roofline(wl, prob, apply_prec, store_prec, step_ms, custom):
    """Roofline of the dominant kernel = the per-step fused operator + recurrence launch(es)."""
    peaks = load_peaks()
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    bf16_peak = peaks.get("bf16_tflops", 1590.0)
    peak_src = "MEASURED_PEAKS.json" if peaks else "fallback (B200_PROFILING.md)"
    m, N = prob["m"], prob["block"]
    sb = 8 if store_prec == "fp64" else 4
    if wl in ("c1", "c2"):
        flops = 2.0 * m * m * N
        tf = flops / (step_ms * 1e-3) / 1e12
        if apply_prec in ("tf32", "bf16"):
            ratio = 0.5 if apply_prec == "tf32" else 1.0
            roof = {"bound": "tensor", "achieved": tf, "peak": bf16_peak * ratio, "unit": "TFLOP/s",
                    "frac": tf / (bf16_peak * ratio), "kernel": "dense step (operator apply + recurrence epilogue)",
                    "peak_source": peak_src + " bf16 burst x %.1f (nominal TF32/BF16 ratio)" % ratio}
        else:
            peak = 37.0 if apply_prec == "fp64" else 75.0
            roof = {"bound": "alu", "achieved": tf, "peak": peak, "unit": "TFLOP/s", "frac": tf / peak,
                    "kernel": "dense SIMT apply + elementwise step", "peak_source": "nominal"}
    else:
        # algorithmic bytes per step: R_Y, R_X, G read once, R_X written once (+ operator bytes), SURVEY 8(d)
        if wl == "c3":
            opb = prob["vals"].size * 8.0
        else:
            opb = prob["n_cells"] * prob["n_loc"] ** 2 * (2.0 if apply_prec == "bf16" else 4.0)
        byts = 4.0 * m * N * sb + opb
        gbs = byts / (step_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                "kernel": "fused operator + recurrence step" + (" (8 colour launches)" if wl in ("c4", "c5") else ""),
                "peak_source": peak_src, "algorithmic_bytes_per_step": byts}
    roof["step_launch_ms"] = step_ms
    tr, src = load_traffic()
    roof["traffic"] = None if custom else tr.get("%s:%s:%s" % (wl, apply_prec, store_prec))
    roof["traffic_source"] = src if roof["traffic"] is not None else None
    return roof


def time_filter(solver, P, X, ritz, G, p, bounds, steps, warmup, dev, world, restore=None, flush=None):
    """W untimed + K timed rchfsi_filter calls; CUDA events on the launching stream; NVML clocks during the
    timed region.  Returns (ms per call [max over ranks], step-kernel ms per launch set, launches, clocks, units)."""
    import torch
    import torch.distributed as dist
    from paper_2503_22652_b200.sharding import reduce_job
    for _ in range(warmup):
        if restore is not None:
            X.copy_(restore)
        solver.filter(P.METHOD_RCHFSI, X, ritz, G, p, *bounds)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    l0 = solver.launch_count()
    total_ms, step_ms, step_n = 0.0, 0.0, 0
    torch.cuda.synchronize()
    for _ in range(steps):
        if flush is not None:
            flush.zero_()                  # L2 flush between timed iterations (outside the event pair)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        solver.filter(P.METHOD_RCHFSI, X, ritz, G, p, *bounds)
        e1.record()
        ms_k, n_k = solver.last_filter_step_ms()   # synchronises: CUDA events around the p-1 step launches
        total_ms += e0.elapsed_time(e1)
        step_ms += ms_k
        step_n += n_k
    torch.cuda.synchronize()
    launches = solver.launch_count() - l0
    clocks = sampler.finish()
    if world > 1:
        dist.barrier()
    m, N = X.shape
    total_ms, updates = reduce_job(total_ms, float(m) * N * p)
    return total_ms / steps, step_ms / max(1, step_n), int(launches), clocks, updates


def time_e2e(solver, P, Xh, rh, Gh, p, bounds, reps, dev, world):
    """The same filter through rchfsi_filter_host: HOST (pinned) buffers, copies inside the timed region."""
    import torch
    import torch.distributed as dist
    solver.filter_host(P.METHOD_RCHFSI, Xh, rh, Gh, p, *bounds)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(reps):
        solver.filter_host(P.METHOD_RCHFSI, Xh, rh, Gh, p, *bounds)
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0) / reps
    te = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    h2d = Xh.numel() * Xh.element_size() + Gh.numel() * Gh.element_size() + rh.numel() * 8
    return float(te.item()), int(h2d), int(Xh.numel() * 8)


def bench_rotation(dev, m=262144, N=2400, reps=5):
    """Sub-record for the Rayleigh-Ritz rotation X = Y E: rchfsi_rotate on a seeded block, INT8
    tensor-pipe path (default) and cuBLAS dgemm (RCHFSI_RR_SPLIT=0) on the same inputs; FP64-equivalent flops = 2 m N^2.
    The INT8 path does 28 digit-plane products per FP64 product: achieved INT8 rate = 28 x 2 m N^2 ops / time."""
    import torch
    import paper_2503_22652_b200 as P
    g = torch.Generator(device=dev).manual_seed(11)
    Y0 = torch.randn((m, N), dtype=torch.float64, device=dev, generator=g)
    E = torch.linalg.qr(torch.randn((N, N), dtype=torch.float64, device=dev, generator=g))[0].contiguous()
    ident = dict(kind="csr", rowptr=torch.arange(m + 1, dtype=torch.int64, device=dev),
                 colind=torch.arange(m, dtype=torch.int32, device=dev), vals=torch.ones(m, dtype=torch.float64, device=dev))
    times, outs = {}, {}
    for name, knob in (("int8", None), ("dgemm", "0")):
        old = os.environ.get("RCHFSI_RR_SPLIT")
        if knob is None:
            os.environ.pop("RCHFSI_RR_SPLIT", None)
        else:
            os.environ["RCHFSI_RR_SPLIT"] = knob
        try:
            s = P.Rchfsi(ident, None, None, block_N=N)       # knobs are read when the handle is created
        finally:
            if old is None:
                os.environ.pop("RCHFSI_RR_SPLIT", None)
            else:
                os.environ["RCHFSI_RR_SPLIT"] = old
        Y = Y0.clone()
        s.rotate(Y, E)
        outs[name] = Y[:512].clone()
        best = None
        sampler = ClockSampler(torch.cuda.current_device())
        sampler.start()
        for _ in range(reps):
            Y.copy_(Y0)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            s.rotate(Y, E)
            e1.record()
            torch.cuda.synchronize()
            t = e0.elapsed_time(e1)
            best = t if best is None else min(best, t)
        clocks = sampler.finish()
        times[name] = (best, clocks)
        s.close()
        del Y
    peaks = load_peaks()
    bf16 = peaks.get("bf16_tflops", 1590.0)
    flops = 2.0 * m * N * N
    ms = times["int8"][0]
    dev_max = float((outs["int8"] - outs["dgemm"]).abs().max() / outs["dgemm"].abs().max())
    return {"metric": "Rayleigh-Ritz rotation X = Y E, FP64-equivalent TFLOP/s", "value": flops / (ms * 1e-3) / 1e12, "unit": "TFLOP/s",
            "ms": ms, "dgemm_ms": times["dgemm"][0], "dgemm_value": flops / (times["dgemm"][0] * 1e-3) / 1e12,
            "speedup_vs_dgemm": times["dgemm"][0] / ms, "max_rel_dev_vs_dgemm": dev_max, "dtype": "int8 digits -> f64",
            "config": {"workload": "rotation of a seeded %d x %d block by a %d x %d orthogonal matrix" % (m, N, N, N)},
            "clocks": times["int8"][1],
            "roofline": {"bound": "tensor", "achieved": 28.0 * flops / (ms * 1e-3) / 1e12, "peak": 2.0 * bf16, "unit": "TOP/s",
                         "frac": 28.0 * flops / (ms * 1e-3) / 1e12 / (2.0 * bf16),
                         "kernel": "i8w_kernel<0> (tcgen05.mma kind::i8, 28 digit-plane products per FP64 product)",
                         "peak_source": "MEASURED_PEAKS.json bf16 burst x 2 (nominal INT8/BF16 ratio)", "traffic": None}}


def bench_resident(key, apply_prec, store_prec, steps, warmup, dev, rank, world, want_e2e, want_cpu, want_solve, args):
    """configs[0..3]: inputs of Alg. 3 (B-orthonormal X, Ritz values, G) from one rchfsi_rayleigh_ritz on the seeded
    start block; filter timed with the inputs resident in HBM, L2 flushed between timed calls."""
    import torch
    import paper_2503_22652_b200 as P
    wl = WORKLOADS[key]
    prob, b = make_problem(key)
    m, N, p, nw = prob["m"], prob["block"], prob["degree"], prob["n_wanted"]
    As, Bs, dinv = P.upload_problem(prob, device=dev)
    noise = dict(noise_eps=prob.get("noise_eps", 0.0), noise_seed=1234) if key == "c1" else {}
    solver = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec, **noise)
    X0 = prob.get("X0")
    if X0 is None:
        X0 = workloads.start_block(m, N, prob.get("x0_seed", 7) + rank)
    X = torch.as_tensor(X0, dtype=torch.float64).to(dev)
    ritz, X, G, _ = solver.rayleigh_ritz(X)
    rz = ritz.cpu().numpy()
    lam_max = b[2] if b[2] is not None else fe_lam_max(prob)
    lam_min = b[0] if b[0] is not None else float(rz[0]) - 1e-2 * max(1.0, abs(float(rz[0])))
    lam_T = b[1] if b[1] is not None else float(rz[-1]) + 1e-6
    bounds = (lam_min, lam_T, lam_max)
    Xwork = X.clone()
    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2
    ms, step_ms, launches, clocks, updates = time_filter(solver, P, Xwork, ritz, G, p, bounds, steps, warmup, dev, world,
                                                         restore=X, flush=flush)
    rec = {"value": updates / (ms * 1e-3), "unit": UNIT, "steps": steps, "warmup": warmup, "ms_per_step": ms,
           "dtype": DTYPE[apply_prec],
           "config": {"workload": wl["name"], "m": m, "block_N": N, "degree": p, "apply_prec": apply_prec,
                      "store_prec": store_prec, "l2": "flushed between timed filter calls (512 MiB memset)",
                      "parallelism": "column shards x%d (operator replicated, no collective)" % world},
           "clocks": clocks, "gpu_launches": launches,
           "roofline": roofline(key, prob, apply_prec, store_prec, step_ms, FE_CELLS is not None or BLOCK is not None)}
    del flush
    if want_e2e:
        Xh = torch.empty((m, N), dtype=torch.float64, pin_memory=True)
        Xh.copy_(X)
        Gh = torch.empty((m, N), dtype=torch.float64, pin_memory=True)
        Gh.copy_(G)
        rh = ritz.cpu().pin_memory()
        e2e_ms, h2d, d2h = time_e2e(solver, P, Xh, rh, Gh, p, bounds, max(1, min(steps, 5)), dev, world)
        rec["e2e"] = {"value": updates / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                      "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms,
                      "pcie_floor_ms": 1e3 * max(h2d / 50e9, d2h / 57e9)}
        del Xh, Gh
    solver.close()
    if want_solve and rank == 0:
        Xs = torch.as_tensor(X0, dtype=torch.float64).to(dev)
        so = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec,
                      adaptive_bounds=(key != "c1"), **noise)
        t0 = time.perf_counter()
        meth = P.METHOD_RCHFSI if args.solve_method == "rchfsi" else P.METHOD_CHFSI
        r = so.solve(meth, Xs, nw, p, lam_min, lam_T, lam_max, tol=1e-8, max_iter=args.solve_iters)
        rec["solve"] = {"method": args.solve_method, "final_residual": float(r["resnorm"][:nw].max()),
                        "iters": int(r["iters"]), "converged": bool(r["converged"]),
                        "seconds": time.perf_counter() - t0, "history": [float(x) for x in r["history"]]}
        so.close()
        del Xs
    if want_cpu and rank == 0:
        cols, deg = CPU_SAMPLE[key]
        v, desc, _ = oracle_sample_time(prob, p, bounds, cols, deg, inputs=(X.cpu().numpy(), rz, G.cpu().numpy()))
        rec["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": desc}
    del X, G, Xwork, solver, As, Bs, dinv
    torch.cuda.empty_cache()
    return rec


def certify_with_oracle(prob, Xd, evals, nw, n_cols=10, seed=77):
    """FP64 residual ||A x - eps B x||_2 and B-norm of sampled returned pairs computed with the
    ORACLE's operators (oracle/chfsi_oracle.py FeOperator, numpy) on the host -- independent of the library's own
    FP64 apply.  A residual <= tau certifies an eigenvalue within tau / sqrt(lam_min(B)) of eps."""
    import torch
    from oracle import chfsi_oracle as orc
    A, B, _ = orc.operators_from_workload(prob)
    rng = np.random.default_rng(seed)
    cols = np.unique(np.concatenate(([0, nw - 1], rng.integers(0, nw, n_cols - 2))))
    Xc = Xd[:, torch.as_tensor(cols, device=Xd.device)].cpu().numpy()
    ev = np.asarray(evals)[cols]
    AX, BX = A.apply(Xc), B.apply(Xc)
    res = np.linalg.norm(AX - BX * ev[None, :], axis=0)
    gram = Xc.T @ BX
    return {"columns": [int(c) for c in cols], "oracle_residual_max": float(res.max()),
            "oracle_borth_err": float(np.abs(gram - np.eye(len(cols))).max()),
            "oracle_rayleigh_quotient_err": float(np.abs(np.diag(Xc.T @ AX) / np.diag(gram) - ev).max())}


def bench_c5(args, dev, rank, world, steps, warmup, apply_prec, store_prec):
    """configs[4] at full size is a memory plan: X FP64 58.5 GB + G FP32 29.3 GB (caller-owned, read in
    place) + R_X, R_Y FP32 58.5 GB + operator copies.  The inputs of Alg. 3 for the timed filter are seeded synthetic
    blocks generated on the device (the filter is defined for any X, Lambda, G)."""
    import torch
    import paper_2503_22652_b200 as P
    wl = WORKLOADS["c5"]
    prob, _ = make_problem("c5")
    m, N, p, nw = prob["m"], prob["block"], prob["degree"], prob["n_wanted"]
    As, Bs, dinv = P.upload_problem(prob, device=dev)
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
    ms, step_ms, launches, clocks, updates = time_filter(solver, P, X, ritz, G, p, bounds, steps, warmup, dev, world)
    finite = bool(torch.isfinite(X[::4096]).all().item())
    rec = {"value": updates / (ms * 1e-3), "unit": UNIT, "steps": steps, "warmup": warmup, "ms_per_step": ms,
           "dtype": DTYPE[apply_prec],
           "config": {"workload": wl["name"], "m": m, "block_N": N, "degree": p, "apply_prec": apply_prec,
                      "store_prec": store_prec, "l2": "inputs (176 GB resident) far larger than L2",
                      "parallelism": "column shards x%d (operator replicated, no collective)" % world,
                      "device_bytes_torch": int(torch.cuda.memory_allocated()), "output_finite": finite},
           "clocks": clocks, "gpu_launches": launches,
           "roofline": roofline("c5", prob, apply_prec, store_prec, step_ms, FE_CELLS is not None or BLOCK is not None)}
    if not args.no_e2e:
        # end to end: the block lives in pinned HOST memory (X FP64 + G FP32 = 88 GB) and goes through the
        # column-chunked pipeline of rchfsi_filter_host; the device-resident inputs are released first
        t0 = time.perf_counter()
        for r0 in range(0, m, 65536):
            X[r0:r0 + 65536].normal_(generator=gen)
        X *= 1.0 / np.sqrt(m)
        Xh = torch.empty((m, N), dtype=torch.float64, pin_memory=True)
        Xh.copy_(X)
        Gh = torch.empty((m, N), dtype=torch.float32, pin_memory=True)
        Gh.copy_(G)
        rh = ritz.cpu().pin_memory()
        del X, G
        torch.cuda.empty_cache()
        t_pin = time.perf_counter() - t0
        e2e_ms, h2d, d2h = time_e2e(solver, P, Xh, rh, Gh, p, bounds, 2, dev, world)
        rec["e2e"] = {"value": updates / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                      "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms,
                      "pcie_floor_ms": 1e3 * max(h2d / 50e9, d2h / 57e9), "host_setup_s": t_pin,
                      "finite": bool(torch.isfinite(Xh[::8192]).all().item())}
        del Xh, Gh
    else:
        rec["e2e"] = None
        del X, G
    solver.close()
    del solver
    torch.cuda.empty_cache()
    if not args.no_solve and rank == 0 and world == 1:
        # full R-ChFSI solve at this size: memory-light mode of the library (chunked Rayleigh-Ritz, FP32 residual
        # block read in place), then the oracle's certificate on sampled wanted pairs
        X = torch.empty((m, N), dtype=torch.float64, device=dev)
        for r0 in range(0, m, 65536):
            X[r0:r0 + 65536].normal_(generator=gen)
        so = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec, adaptive_bounds=True)
        t0 = time.perf_counter()
        r = so.solve(P.METHOD_RCHFSI, X, nw, p, -100.0, 0.0, bounds[2], tol=1e-8, max_iter=args.solve_iters)
        sol = {"final_residual": float(r["resnorm"][:nw].max()), "iters": int(r["iters"]),
               "converged": bool(r["converged"]), "seconds": time.perf_counter() - t0,
               "history": [float(x) for x in r["history"]],
               "evals_first_last_wanted": [float(r["evals"][0]), float(r["evals"][nw - 1])],
               "device_bytes_torch": int(torch.cuda.memory_allocated())}
        so.close()
        t0 = time.perf_counter()
        sol.update(certify_with_oracle(prob, X, r["evals"], nw))
        sol["certify_seconds"] = time.perf_counter() - t0
        sol["certified"] = bool(sol["converged"] and sol["oracle_residual_max"] <= 1e-8 * 1.01
                                and sol["oracle_borth_err"] <= 1e-8)
        # split of the solve's wall time, derived: Alg. 1 runs one Rayleigh-Ritz, then iters x (filter + Rayleigh-Ritz)
        sol["filter_seconds_each"] = rec["ms_per_step"] * 1e-3
        sol["rayleigh_ritz_seconds_each_derived"] = max(0.0, sol["seconds"] - sol["iters"] * rec["ms_per_step"] * 1e-3) / (sol["iters"] + 1)
        rec["solve"] = sol
        del X
        torch.cuda.empty_cache()
    if not args.no_cpu_baseline and rank == 0:
        cols, deg = CPU_SAMPLE["c5"]
        v, desc, _ = oracle_sample_time(prob, p, bounds, cols, deg)
        rec["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": desc}
    del As, Bs, dinv
    torch.cuda.empty_cache()
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5", choices=sorted(WORKLOADS))
    ap.add_argument("--apply-prec", default=None)
    ap.add_argument("--store-prec", default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-solve", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the sub-records of the other kernel claims")
    ap.add_argument("--solve", action="store_true", help="c4: also run rchfsi_solve (about half a minute)")
    ap.add_argument("--solve-method", default="rchfsi", choices=["rchfsi", "chfsi"],
                    help="method of the extra solve (chfsi = Algorithm 2 with the same kernels, the paper's comparator)")
    ap.add_argument("--solve-iters", type=int, default=60)
    ap.add_argument("--profile-run", action="store_true",
                    help="exit 0 even when a deliberately truncated solve (--solve-iters) is not certified: for ncu passes")
    ap.add_argument("--fe-cells", type=int, default=None, help="c4/c5: cells per direction (profiling a smaller mesh)")
    ap.add_argument("--block", type=int, default=None, help="override the block width N (profiling)")
    args = ap.parse_args()
    global FE_CELLS, BLOCK
    FE_CELLS, BLOCK = args.fe_cells, args.block
    if args.impl == "reference":
        run_reference(args)
        return
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist

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
    t_start = time.perf_counter()
    if args.workload == "c5":
        rec = bench_c5(args, dev, rank, world, args.steps, args.warmup, apply_prec, store_prec)
    else:
        want_solve = (not args.no_solve) and (args.workload in ("c1", "c2", "c3") or args.solve)
        rec = bench_resident(args.workload, apply_prec, store_prec, args.steps, args.warmup, dev, rank, world,
                             not args.no_e2e, not args.no_cpu_baseline, want_solve, args)
    out = {"metric": METRIC, "value": rec.pop("value"), "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": rec.pop("ms_per_step"), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": rec.pop("dtype"), "data": "synthetic"}
    rec.pop("steps", None)
    rec.pop("warmup", None)
    rec.pop("unit", None)
    out.update(rec)
    if args.workload == "c5" and not args.no_also and world == 1 and FE_CELLS is None and BLOCK is None:
        also = {}
        for key, wkey, ap_, sp_, kmax in ALSO:
            try:
                also[key] = bench_resident(wkey, ap_, sp_, min(args.steps, kmax), 3, dev, rank, world, wkey != "c2",
                                           False, False, args)
            except Exception as exc:     # one failing sub-record must not lose the line
                also[key] = {"error": "%s: %s" % (type(exc).__name__, exc)}
                torch.cuda.empty_cache()
        try:
            also["rr_rotation_int8"] = bench_rotation(dev)
        except Exception as exc:
            also["rr_rotation_int8"] = {"error": "%s: %s" % (type(exc).__name__, exc)}
        torch.cuda.empty_cache()
        out["also"] = also
    out["wall_s_total"] = time.perf_counter() - t_start
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    if rank == 0 and isinstance(out.get("solve"), dict) and out["solve"].get("certified") is False:
        sys.stderr.write("bench.py: the configs[4] solve is NOT certified by the oracle: %s\n" % json.dumps(out["solve"]))
        if not args.profile_run:
            sys.exit(3)


if __name__ == "__main__":
    main()
