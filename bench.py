"""bench.py -- headline benchmark of the B200-native TDVP hot path (BASELINE.json metric:
"H_eff.A applies/s and TDVP-PS step time at M=128; % FP64 tensor-core peak").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" = APPLIES_PER_STEP H_eff applies of BASELINE.json configs[1] at
M = 128 (d = 10, D_W = 20, 6000 non-zeros of W), each on the next of N_SETS resident input sets
(total > L2, so L, A, R are L2-cold), through the C ABI (tdvp_apply_heff).  `value` = applies/s with
inputs resident in HBM; `e2e` = the same through tdvp_apply_heff_host (HOST buffers, h2d + d2h
inside the timed region).  Also reported on the same JSON line: the M sweep, the environment update
(a4), one TDVP-PS step (a5-a8, a10) of the M = 128 FMO-like chain (configs[3]), the roofline of the
dominant kernel (DMMA complex GEMM) from live CUDA-event brackets, and the oracle timed on the
host cores (cpu_baseline).  Multi-GPU: the path does not shard -- "replicas only":
every rank runs the same workload, `value` is the sum over ranks.
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

import synthetic_inputs as si  # noqa: E402

M_HEADLINE, D_PHYS, D_W, NNZ = 128, 10, 20, 6000
APPLIES_PER_STEP = 24
N_SETS = 12                      # 12 x (L 5.2 + A 2.6 + R 5.2 + out 2.6 MB) = 188 MB > 126 MB L2
METRIC, UNIT = "heff_applies_per_s_M128", "applies/s"
WORKLOAD = "configs[1]: isolated H_eff.A, complex128, M=128, d=10, D_W=20, W 15% dense (6000 nnz)"


def heff_flops(M, d=D_PHYS, Dw=D_W, nnz=NNZ):
    """Algorithmic flops of one apply: two GEMM stages 8 M^3 D_W d each + W stage 8 M^2 nnz."""
    return 16.0 * M ** 3 * Dw * d + 8.0 * M ** 2 * nnz


def gemm_stage_flops(M, d=D_PHYS, Dw=D_W):
    return 8.0 * M ** 3 * Dw * d


def heff_executed_flops(M, products, d=D_PHYS, Dw=D_W, nnz=NNZ):
    """Flops the kernels EXECUTE for one apply: the GEMM stages form a complex multiply-add from
    `products` real DMMA products (2 flops each: 6 or 8 per complex multiply-add), the W stage from 4 DFMA."""
    return 2.0 * products * 2.0 * M ** 3 * Dw * d + 8.0 * M ** 2 * nnz


def site_apply_flops(Ml, Mr, d, Dl, Dr, nnz):
    """(GEMM-stage, W-stage) algorithmic flops of one H_eff apply / environment update of a site
    (8 flops per complex multiply-add)."""
    return 8.0 * (Ml * Ml * Dl * d * Mr + Ml * d * Dr * Mr * Mr), 8.0 * Ml * Mr * nnz


def qr_flops(rows, cols):
    """Householder QR of a complex rows x cols matrix plus forming Q: 2 x (8 rows cols^2 - 8/3 cols^3)."""
    return 2.0 * (8.0 * rows * cols * cols - 8.0 / 3.0 * cols ** 3)


def ps_step_flops(mpo, mps, k):
    """Algorithmic flops of one TDVP-PS step (Eq. 42) of THIS chain, from its actual M_i, D_W,i and
    nnz(W_i), with the formula of SURVEY.md 8(a) a8: (2N-1) k H_eff applies, 2(N-1) environment updates,
    2(N-1) k bond applies, 2(N-1) QR gauge moves + absorbs, and the Krylov vector work (two Gram-Schmidt
    passes over j+1 vectors per iteration + the final combination).  Returns (gemm, wstage, other)."""
    n = len(mps)
    gemm = wst = other = 0.0
    for i in range(n):
        Ml, d, Mr = mps[i].shape
        Dl, Dr = mpo[i].shape[0], mpo[i].shape[3]
        g, w = site_apply_flops(Ml, Mr, d, Dl, Dr, int(np.count_nonzero(mpo[i])))
        n_exp = 1 if i == n - 1 else 2
        gemm += n_exp * k * g
        wst += n_exp * k * w
        nvec = Ml * d * Mr
        other += n_exp * (8.0 * nvec * (k * (k + 1) + k))          # 2 passes x (dot + axpy) x sum_j (j+1), + combine
        if i < n - 1:                                             # forward QR + left environment, Eq. 9, 30-32
            gemm += g
            wst += w
            other += qr_flops(Ml * d, Mr)
        if i > 0:                                                 # backward RQ + right environment
            gemm += g
            wst += w
            other += qr_flops(d * Mr, Ml)
            gemm += 2 * k * 8.0 * (Ml * Ml * Dl * Ml + Ml * Dl * Ml * Ml)   # bond applies of bond i, both sweeps (Eq. 44)
            gemm += 2 * 8.0 * Ml * Ml * d * Mr                                # absorbs C = D B, C = A D
            other += 2 * (8.0 * Ml * Ml * (k * (k + 1) + k))
    return gemm, wst, other


def cmf_step_flops(mpo, mps, k, n_sub):
    """Algorithmic flops of one second-order CMF step: two mean-field builds (N-1 left
    and N-1 right environments, N-1 centre-form GEMMs; SVDs counted as QR + 8 Ml^3 x 10 sweeps of Jacobi),
    local RK4 propagation with ceil(n_sub/2) + n_sub sub-steps x 4 right-hand sides per site (one H_eff apply +
    four (rows x Jr x Jr) GEMMs each), and two Krylov exponentials at the last site."""
    n = len(mps)
    gemm = wst = other = 0.0
    nrhs = 4 * ((n_sub + 1) // 2 + n_sub)
    for i in range(n):
        Ml, d, Mr = mps[i].shape
        Dl, Dr = mpo[i].shape[0], mpo[i].shape[3]
        g, w = site_apply_flops(Ml, Mr, d, Dl, Dr, int(np.count_nonzero(mpo[i])))
        if i < n - 1:
            gemm += 2 * g + nrhs * (g + 4 * 8.0 * Ml * d * Mr * Mr)
            wst += 2 * w + nrhs * w
        else:
            gemm += 2 * k * g
            wst += 2 * k * w
        if i > 0:
            gemm += 2 * (g + 8.0 * Ml * Ml * d * Mr)
            wst += 2 * w
            other += 2 * (qr_flops(d * Mr, Ml) + 80.0 * Ml ** 3)
    return gemm, wst, other


def time_cublas_fp64(torch, seconds=4.0):
    """cuBLAS FP64 ceilings of THIS box, measured in this run (SURVEY.md 8(d) "Peaks to divide by"): they are
    DENOMINATORS only -- torch.matmul is never on the hot path.  ZGEMM 4096^3 (8 flops per complex multiply-add)
    and DGEMM 8192^3, best of 10 (burst) and back to back for `seconds` (sustained)."""
    out = {}
    for name, n, dtype, flops in (("zgemm", 4096, torch.complex128, 8.0 * 4096 ** 3), ("dgemm", 8192, torch.float64, 2.0 * 8192 ** 3)):
        a = torch.randn(n, n, dtype=dtype, device="cuda")
        b = torch.randn(n, n, dtype=dtype, device="cuda")
        c = torch.empty_like(a)
        for _ in range(2):
            torch.matmul(a, b, out=c)
        best = 1e30
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(10):
            e0.record(); torch.matmul(a, b, out=c); e1.record(); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        reps = max(3, int(seconds * 1e3 / best))
        e0.record()
        for _ in range(reps):
            torch.matmul(a, b, out=c)
        e1.record(); torch.cuda.synchronize()
        out[name] = {"n": n, "burst_tflops": flops / (best * 1e-3) / 1e12,
                     "sustained_tflops": flops * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12, "sustained_s": e0.elapsed_time(e1) * 1e-3}
        del a, b, c
    torch.cuda.empty_cache()
    return out


def committed_traffic(kernel, M):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` at bond dimension M from the
    committed ncu --set full summary profiles/kernel_traffic.csv (columns: kernel, M, dram_bytes_per_launch,
    capture); None if there is no such row.  bench.py never runs under ncu, so this is the only place the
    number can come from; the csv names the capture it was read from."""
    path = os.path.join(ROOT, "profiles", "kernel_traffic.csv")
    try:
        rows = [l.strip().split(",") for l in open(path) if l.strip() and not l.startswith("#")]
    except OSError:
        return None, None
    best = (None, None)
    for r in rows[1:]:
        if len(r) >= 4 and r[0] == kernel and int(r[1]) == M:
            best = (float(r[2]), r[3])                  # later rows (later rounds) win
    return best


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_cores():
    try:
        from threadpoolctl import threadpool_info
        n = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
        return int(n)
    except Exception:
        return os.cpu_count() or 1


def time_oracle_heff(M, min_seconds=10.0, max_applies=200):
    """The oracle's heff, as it stands, on the host cores: applies/s over a bounded sample."""
    from oracle import contractions as oc
    L, W, A, R = si.microbench_tensors(M)
    oc.heff(L, W, A, R)
    n, t0 = 0, time.perf_counter()
    while True:
        oc.heff(L, W, A, R)
        n += 1
        el = time.perf_counter() - t0
        if el >= min_seconds or n >= max_applies:
            break
    return n / el, n, el


def run_reference(args):
    """--impl reference: the oracle (oracle/contractions.py heff) on the host cores, same metric
    and config; each step is ONE apply (a bounded sample of the APPLIES_PER_STEP-apply step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import contractions as oc
    L, W, A, R = si.microbench_tensors(M_HEADLINE)
    for _ in range(max(1, min(args.warmup, 3))):
        oc.heff(L, W, A, R)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oc.heff(L, W, A, R)
    el = time.perf_counter() - t0
    val = args.steps / el
    cores = oracle_cores()
    sample = "1 oracle heff apply per step (of the %d-apply step), %d steps, numpy tensordot" % (APPLIES_PER_STEP, args.steps)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "c128", "data": "synthetic", "config": {"workload": WORKLOAD},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def make_sets(torch, M, n_sets):
    """n_sets independent resident input sets of configs[1] at bond dimension M (seeded)."""
    sets = []
    for s in range(n_sets):
        L, W, A, R = si.microbench_tensors(M, seed=1000 + M + 7919 * s)
        sets.append([torch.from_numpy(x).cuda() for x in (L, W, A, R)] +
                    [torch.empty((M, D_PHYS, M), dtype=torch.complex128, device="cuda")])
    return sets


def time_applies(torch, T, ctx, sets, n_applies):
    """CUDA-event time (ms) of n_applies back-to-back calls on torch's current stream."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(n_applies):
        L, W, A, R, out = sets[i % len(sets)]
        T.tdvp_apply_heff(L, W, A, R, out=out, handle=ctx)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def sweep_point(torch, T, M, peak_tflops):
    """applies/s and fraction of the FP64 tensor peak at one M of the configs[1] sweep."""
    per_set = 16.0 * M * M * (2 * D_W + 2 * D_PHYS)
    n_sets = int(max(2, min(16, np.ceil(1.5 * 126e6 / per_set)))) if M < 512 else 2
    sets = make_sets(torch, M, n_sets)
    ctx = T.tdvp_create_context()
    n = int(max(4, min(200, 2e11 / heff_flops(M))))
    time_applies(torch, T, ctx, sets, max(3, n // 4))
    ms = time_applies(torch, T, ctx, sets, n)
    env_out = torch.empty((M, D_W, M), dtype=torch.complex128, device="cuda")
    for _ in range(3):
        T.tdvp_update_env(0, sets[0][0], sets[0][1], sets[0][2], env_out=env_out, handle=ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(n):
        s = sets[i % len(sets)]
        T.tdvp_update_env(0, s[0], s[1], s[2], env_out=env_out, handle=ctx)
    e1.record()
    torch.cuda.synchronize()
    ms_env = e0.elapsed_time(e1)
    ctx.close()
    aps = n / (ms * 1e-3)
    products = T.tdvp_get_gemm_products()
    # effective_tflops counts ALGORITHMIC flops (8 per complex multiply-add) and may exceed the pipe's peak when
    # the GEMM stages run the 3-product form; frac_fp64_tensor_peak counts the flops actually EXECUTED: <= 1
    return {"M": M, "applies_per_s": aps, "us_per_apply": 1e3 * ms / n, "effective_tflops": aps * heff_flops(M) / 1e12,
            "executed_tflops": aps * heff_executed_flops(M, products) / 1e12,
            "frac_fp64_tensor_peak": aps * heff_executed_flops(M, products) / 1e12 / peak_tflops,
            "env_updates_per_s": n / (ms_env * 1e-3), "input_sets": n_sets}


def build_chain(name, M=None):
    """MPO (built by the library's own host-side builder, tdvp_build_vibronic_mpo: SURVEY.md A21) and the
    seeded delta-padded initial MPS of one of BASELINE.json's chain configs."""
    import dataclasses
    import paper_1907_12044_b200 as T
    cfg = si.CONFIGS[name]
    if M is not None:
        cfg = dataclasses.replace(cfg, M=M)
    params = si.draw_vibronic_params(cfg)
    mpo = T.tdvp_build_vibronic_mpo(params.E, params.J, params.omega, params.S, params.n_ph, params.layout)
    dims = si.site_dims(params)
    mps = si.padded_product_mps(dims, si.initial_occupations(params), cfg.M, cfg.pad_seed, cfg.delta, cfg.delta_seed)
    return cfg, mpo, mps


def rank_max(x, world, device):
    """Replicas only: the ranks share nothing but the clock -- the step time of the job
    is the MAX over ranks (all-reduce on `device`: "cuda" under NCCL, "cpu" under gloo in the tests)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(units_per_rank, world, ms_max):
    """Whole-job throughput: the units ALL ranks processed divided by the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_1907_12044_b200 as T
    T.library_path()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return rank_max(x, world, "cuda")

    peak = T.tdvp_probe_fp64_tensor_peak(20000)        # DMMA issue-rate ceiling, measured live
    M = M_HEADLINE
    sets = make_sets(torch, M, N_SETS)
    ctx = T.tdvp_create_context()
    launches0 = T.tdvp_launch_count()

    # ---- resident-input arm: W warm-up steps, then exactly K timed steps ----
    for _ in range(args.warmup):
        time_applies(torch, T, ctx, sets, APPLIES_PER_STEP)
    sampler = ClockSampler(local)
    sampler.start()
    T.tdvp_profile_enable(True)
    T.tdvp_profile_read()
    barrier()
    l0 = T.tdvp_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for s in range(args.steps):
        for i in range(APPLIES_PER_STEP):
            L, W, A, R, out = sets[(s * APPLIES_PER_STEP + i) % N_SETS]
            T.tdvp_apply_heff(L, W, A, R, out=out, handle=ctx)
    e1.record()
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    gpu_launches = T.tdvp_launch_count() - l0
    prof = T.tdvp_profile_read()
    T.tdvp_profile_enable(False)
    clocks = sampler.stop()
    n_applies = args.steps * APPLIES_PER_STEP
    value = job_value(n_applies, world, ms_total)

    # ---- roofline of the dominant kernel (DMMA complex GEMM): live event brackets above ----
    zg_ms, zg_n = prof["zgemm"]
    ws_ms, ws_n = prof["wstage"]
    flops_per_launch = gemm_stage_flops(M)             # each of the 2 GEMM launches of an apply
    achieved = flops_per_launch / (zg_ms / max(zg_n, 1) * 1e-3) / 1e12 if zg_n else None
    products = T.tdvp_get_gemm_products()
    traffic, traffic_src = committed_traffic("zgemm_kernel", M)
    roofline = {"bound": "tensor", "kernel": "zgemm_kernel (FP64 DMMA m8n8k4, complex128)",
                "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": (achieved / peak) if achieved else None,
                # "achieved" counts ALGORITHMIC flops (8 per complex multiply-add); the kernel forms
                # the complex product from `gemm_products` real DMMA products (3 by default: 6 executed flops per
                # complex multiply-add), so the share of the DMMA pipe it keeps busy is frac * products / 4
                "gemm_products": products,
                "dmma_pipe_frac": (achieved / peak * products / 4.0) if achieved else None,
                # dram__bytes_read.sum + dram__bytes_write.sum per launch, read from the committed ncu --set full
                # summary (profiles/kernel_traffic.csv names the capture); null if no capture of this kernel at this M
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "tdvp_probe_fp64_tensor_peak: DMMA m8n8k4 issue rate measured in this run (MEASURED_PEAKS.json has "
                               "no FP64 figure); the cuBLAS ZGEMM / DGEMM rates of this box, measured in this run, are beside it",
                "flops_per_launch": flops_per_launch, "avg_launch_us": 1e3 * zg_ms / max(zg_n, 1), "launches": zg_n,
                "share_of_step": {"zgemm": zg_ms / ms_total, "wstage": ws_ms / ms_total},
                "wstage": {"bound": "hbm", "note": "algorithmic bytes = one read of T1 + one write of T2; ncu shows the kernel bound by "
                                                  "shared-memory (LSU) wavefronts, not by HBM (profiles/r01e_summary.md)",
                           "algorithmic_bytes": 2 * 16.0 * M * M * D_W * D_PHYS,
                           "achieved_gbs": (2 * 16.0 * M * M * D_W * D_PHYS / (ws_ms / max(ws_n, 1) * 1e-3) / 1e9) if ws_n else None,
                           "avg_launch_us": 1e3 * ws_ms / max(ws_n, 1)}}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        roofline["wstage"]["peak_gbs"] = peaks.get("hbm_gbs")
        if roofline["wstage"]["achieved_gbs"] and peaks.get("hbm_gbs"):
            roofline["wstage"]["frac"] = roofline["wstage"]["achieved_gbs"] / peaks["hbm_gbs"]
    except OSError:
        roofline["wstage"]["peak_gbs"] = 6650.0
        roofline["wstage"]["peak_source"] = "fallback"

    # ---- end-to-end arm: HOST (pinned) buffers through tdvp_apply_heff_host ----
    hsets = []
    for s in range(3):
        arrs = []
        for x in si.microbench_tensors(M, seed=1000 + M + 7919 * s) + (np.empty((M, D_PHYS, M), np.complex128),):
            t = torch.empty(x.shape, dtype=torch.complex128).pin_memory()
            t.numpy()[...] = x
            arrs.append(t.numpy())
        hsets.append(arrs)
    h2d = sum(a.nbytes for a in hsets[0][:4])
    d2h = hsets[0][4].nbytes
    e2e_applies = max(4, min(n_applies, 40))
    for i in range(3):
        T.tdvp_apply_heff_host(*hsets[i % 3], handle=ctx)
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_applies):
        T.tdvp_apply_heff_host(*hsets[i % 3], handle=ctx)
    torch.cuda.synchronize()
    el = max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * e2e_applies / el, "unit": UNIT, "h2d_bytes_per_step": h2d * APPLIES_PER_STEP,
           "d2h_bytes_per_step": d2h * APPLIES_PER_STEP, "applies_timed": e2e_applies,
           "api": "tdvp_apply_heff_host (pinned host buffers; h2d L,W,A,R + kernels + d2h out per apply)"}
    ctx.close()
    del sets
    torch.cuda.empty_cache()

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_total / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
           "config": {"workload": WORKLOAD, "applies_per_step": APPLIES_PER_STEP, "input_sets": N_SETS,
                      "l2": "inputs rotate over %d resident sets (188 MB > 126 MB L2); T1/T2 intermediates 52 MB each" % N_SETS,
                      "multi_gpu": "replicas only (SURVEY.md 8(e))", "seed": "1000+M+7919*set"},
           "us_per_apply": 1e3 * ms_total / n_applies,
           "effective_tflops": value / world * heff_flops(M) / 1e12,
           "executed_tflops": value / world * heff_executed_flops(M, products) / 1e12,
           "frac_fp64_tensor_peak": value / world * heff_executed_flops(M, products) / 1e12 / peak,
           "flop_convention": "frac_fp64_tensor_peak divides the flops the kernels EXECUTE (GEMM stages: 2 x gemm_products per complex "
                              "multiply-add, 6 with the default 3-product form; W stage: 8) by the measured DMMA peak: pipe utilisation, "
                              "never above 1.  effective_tflops counts ALGORITHMIC flops (8 per complex multiply-add, SURVEY.md 8(d)), as "
                              "does roofline.achieved (the contract's definition); roofline.dmma_pipe_frac is its executed counterpart",
           "roofline": roofline, "e2e": e2e, "gpu_launches": int(gpu_launches), "clocks": clocks}

    if rank == 0 and not args.no_extras:
        # cuBLAS FP64 ceilings of this box (denominators only)
        cub = time_cublas_fp64(torch)
        out["roofline"]["peak_cublas_zgemm"] = cub["zgemm"]
        out["roofline"]["peak_cublas_dgemm"] = cub["dgemm"]
        # the same resident-input loop with the complex product from FOUR real DMMA products (reading c15)
        sets = make_sets(torch, M, N_SETS)
        ctx = T.tdvp_create_context()
        T.tdvp_set_gemm_products(4)
        try:
            time_applies(torch, T, ctx, sets, APPLIES_PER_STEP)
            ms4 = time_applies(torch, T, ctx, sets, 4 * APPLIES_PER_STEP)
        finally:
            T.tdvp_set_gemm_products(3)
        out["gemm_products_4"] = {"applies_per_s": 4 * APPLIES_PER_STEP / (ms4 * 1e-3), "us_per_apply": 1e3 * ms4 / (4 * APPLIES_PER_STEP),
                                  "frac_fp64_tensor_peak": 4 * APPLIES_PER_STEP / (ms4 * 1e-3) * heff_executed_flops(M, 4) / 1e12 / peak}
        ctx.close()
        del sets
        torch.cuda.empty_cache()
        # what non-tensor instructions cost the FP64 tensor pipe: TFLOP/s with F
        # integer instructions issued after every DMMA, two CTAs of four warps per SM
        out["dmma_issue_probe_tflops"] = {str(f): T.tdvp_probe_dmma_issue(f, 4000) for f in (0, 1, 2, 4, 8, 16)}
        # M sweep of configs[1]
        out["sweep"] = [sweep_point(torch, T, m, peak) for m in (32, 64, 128, 256, 512)]
        torch.cuda.empty_cache()
        # one TDVP-PS step of the FMO-like chain at M = 128 (configs[3]; k = 10, dt = 5 fs)
        cfg, mpo, mps = build_chain("fmo128")
        ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim))
        for _ in range(2):
            ch.tdvp_step_ps(cfg.dt_fs)
        ch.tdvp_sync()
        l0 = T.tdvp_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        n_ps = 3
        for _ in range(n_ps):
            ch.tdvp_step_ps(cfg.dt_fs)
        e1.record()
        ch.tdvp_sync()
        torch.cuda.synchronize()
        nrm, en = ch.tdvp_norm_energy()
        fg, fw, fo = ps_step_flops(mpo, mps, cfg.krylov_dim)
        ps_ms = e0.elapsed_time(e1) / n_ps
        out["ps_step"] = {"workload": "configs[3]: FMO-like chain, 71 sites, M=128, D_W<=9 (real MPO), k=10, dt=5 fs, CUDA graph",
                          "ms_per_step": ps_ms, "steps_timed": n_ps,
                          # algorithmic flops of one step of THIS chain (its M_i, D_W,i, nnz(W_i))
                          "flops": {"gemm": fg, "wstage": fw, "qr_and_vectors": fo, "total": fg + fw + fo},
                          "effective_tflops": (fg + fw + fo) / (ps_ms * 1e-3) / 1e12,
                          "frac_fp64_tensor_peak": (products / 4.0 * fg + fw + fo) / (ps_ms * 1e-3) / 1e12 / peak,
                          "ms_at_peak": (products / 4.0 * fg + fw + fo) / (peak * 1e12) * 1e3,
                          "launches_per_step": (T.tdvp_launch_count() - l0) // n_ps,
                          "norm_sq": nrm, "energy": en, "populations": ch.tdvp_populations(0).tolist()}
        ch.close()
        # phase breakdown of one step (direct enqueue, event brackets per kernel class; the graph replay above is the timed number)
        ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim, flags=T.TDVP_FLAG_NO_GRAPH))
        ch.tdvp_step_ps(cfg.dt_fs)
        ch.tdvp_sync()
        T.tdvp_profile_enable(True)
        T.tdvp_profile_read()
        e0.record()
        ch.tdvp_step_ps(cfg.dt_fs)
        e1.record()
        ch.tdvp_sync()
        torch.cuda.synchronize()
        ph = T.tdvp_profile_read()
        T.tdvp_profile_enable(False)
        out["ps_step"]["no_graph_ms"] = e0.elapsed_time(e1)
        out["ps_step"]["phase_ms"] = {k: round(v[0], 3) for k, v in ph.items()}
        out["ps_step"]["phase_brackets"] = {k: v[1] for k, v in ph.items()}
        ch.close()
        # (f)3: the same step with the adaptive Krylov dimension (device-side rule, cap 40, tol 1e-8): the configured
        # k = 10 is far from converged at this dt, so both are reported side by side
        try:
            KCAP, KTOL = 40, 1e-8
            ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=KCAP, krylov_tol=KTOL))
            ch.tdvp_step_ps(cfg.dt_fs)
            ch.tdvp_sync()
            e0.record()
            for _ in range(2):
                ch.tdvp_step_ps(cfg.dt_fs)
            e1.record()
            ch.tdvp_sync()
            torch.cuda.synchronize()
            nrm, en = ch.tdvp_norm_energy()
            out["ps_step_adaptive_krylov"] = {"krylov_cap": KCAP, "krylov_tol": KTOL, "ms_per_step": e0.elapsed_time(e1) / 2,
                                              "norm_sq": nrm, "energy": en,
                                              "note": "stop at the first j with beta_j |[exp(z T_j) e_1]_j| < tol, decided on the device; "
                                                      "applies after the stop return at once (skip flag)"}
            ch.close()
        except Exception as ex:                      # noqa: BLE001 -- a bench extra must not take the headline down
            out["ps_step_adaptive_krylov"] = {"error": str(ex)}
        # (f)2: the paper's warm-up: 10 P&C-RK4 steps of 80 a.u. from the bare product state, on the
        # device, then compression -- at M = 14 (M_O M <= 128 keeps every SVD on the fast Jacobi path; at M = 128 the
        # compression SVDs are 1152 x 1152: DESIGN.md 6).  Then: the largest Dormand-Prince step h that keeps
        # err_est <= 1e-7 from the WARMED start against the delta-seeded padded start after 5 PS steps (both M = 14)
        try:
            import dataclasses
            M_W, AU = 14, 0.0241888
            cfgw = dataclasses.replace(si.CONFIGS["fmo128"], M=M_W)
            params = si.draw_vibronic_params(cfgw)
            dims = si.site_dims(params)
            prod = []
            for dd, oo in zip(dims, si.initial_occupations(params)):
                a = np.zeros((1, dd, 1), dtype=np.complex128)
                a[0, oo, 0] = 1.0
                prod.append(a)
            t0 = time.perf_counter()
            TAU_W = 20 * AU      # 80 a.u. (the paper's) is outside RK4's stability region on this chain: (n_ph-1) w_max tau = 4.9 > 2.8
            warm = T.tdvp_pc_rk4_warmup(mpo, prod, TAU_W, 10, M_W, M_W)
            warm_s = time.perf_counter() - t0
            H_LIST = [30 * AU, 15 * AU, 5 * AU, 0.05, 0.02, 0.01, 0.004]

            def mu_errs(start_mps, n_ps):
                chw = T.tdvp_create(mpo, start_mps, T.make_options(krylov_dim=cfg.krylov_dim))
                for _ in range(n_ps):
                    chw.tdvp_step_ps(cfg.dt_fs)
                base = chw.tdvp_get_mps()
                errs = {}
                for h in H_LIST:
                    chw.tdvp_set_mps(base, 0)
                    errs["%.4f" % h] = chw.tdvp_step_mu(h, want_err=True)
                chw.close()
                ok = [h for h in H_LIST if np.isfinite(errs["%.4f" % h]) and errs["%.4f" % h] <= 1e-7]
                return errs, (max(ok) if ok else None)

            errs_w, h_w = mu_errs(warm, 0)
            padded = si.padded_product_mps(dims, si.initial_occupations(params), M_W, cfgw.pad_seed, cfgw.delta, cfgw.delta_seed)
            errs_p, h_p = mu_errs(padded, 5)
            out["pc_rk4_warmup"] = {"workload": "configs[3] chain (71 sites), 10 P&C-RK4 steps of 20 a.u. at M_max = %d, compressed to %d" % (M_W, M_W),
                                    "seconds": warm_s, "bonds_max": max(a.shape[2] for a in warm),
                                    "dp5_err_est_by_h_fs": {"warmed": errs_w, "padded_delta_seeded_after_5_ps_steps": errs_p},
                                    "largest_h_fs_with_err_below_1e-7": {"warmed": h_w, "padded": h_p},
                                    "paper_step_range_fs": [5 * AU, 30 * AU]}
        except Exception as ex:                      # noqa: BLE001
            out["pc_rk4_warmup"] = {"error": str(ex)}
        # TDVP-MU on the same chain (configs[3]): five PS steps of warm-up (the MU right-hand side needs
        # full-rank bonds, DESIGN.md c18), then Dormand-Prince steps of h = 0.004 fs: with eps = 1e-10 the
        # right-hand side is stiff (1 / sqrt(eps) = 1e5 on the weakly occupied bonds of this chain), the
        # explicit 5(4) pair is stable up to h ~ 0.02 fs and overflows at 0.1 fs (DESIGN.md c12)
        ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim))
        for _ in range(5):
            ch.tdvp_step_ps(cfg.dt_fs)
        H_MU = 0.004
        ch.tdvp_step_mu(H_MU)
        ch.tdvp_sync()
        T.tdvp_profile_enable(True)
        T.tdvp_profile_read()
        e0.record()
        n_mu = 2
        for _ in range(n_mu):
            err = ch.tdvp_step_mu(H_MU, want_err=True)
        e1.record()
        ch.tdvp_sync()
        torch.cuda.synchronize()
        ph = T.tdvp_profile_read()
        T.tdvp_profile_enable(False)
        nrm, en = ch.tdvp_norm_energy()
        out["mu_step"] = {"workload": "configs[3] chain, 71 sites, M=128: one Dormand-Prince 5(4) step of h = 0.004 fs "
                                      "(7 right-hand sides: SVD + environments + H_eff per site) after 5 PS steps",
                          "ms_per_step": e0.elapsed_time(e1) / n_mu, "steps_timed": n_mu, "err_est": err, "norm_sq": nrm,
                          "energy": en, "phase_ms_per_step": {k: round(v[0] / n_mu, 3) for k, v in ph.items()}}
        # TDVP-MU with constant-mean-field integration from the
        # same state: CMF steps of tau = 0.1 fs, 10 RK4 sub-steps per site (local step 0.01 fs, inside the
        # stability limit the stiff right-hand side sets, see above); SVDs and environments twice per step
        TAU_CMF, NSUB_CMF = 0.1, 10
        ch.tdvp_step_mu_cmf(TAU_CMF, NSUB_CMF)              # (captures the step's CUDA graph)
        ch.tdvp_sync()
        l0 = T.tdvp_launch_count()
        e0.record()
        n_cmf = 2
        for _ in range(n_cmf):
            ch.tdvp_step_mu_cmf(TAU_CMF, NSUB_CMF)          # timed: graph replays
        e1.record()
        ch.tdvp_sync()
        torch.cuda.synchronize()
        cmf_ms = e0.elapsed_time(e1) / n_cmf
        cmf_launches = (T.tdvp_launch_count() - l0) // n_cmf
        nrm, en = ch.tdvp_norm_energy()
        # phase breakdown: one more step with the profiler on, which makes the library enqueue it directly
        # (a replayed graph carries no event brackets); its wall time is reported beside the graph's
        T.tdvp_profile_enable(True)
        T.tdvp_profile_read()
        e0.record()
        ch.tdvp_step_mu_cmf(TAU_CMF, NSUB_CMF)
        e1.record()
        ch.tdvp_sync()
        torch.cuda.synchronize()
        ph = T.tdvp_profile_read()
        T.tdvp_profile_enable(False)
        cmf_direct_ms = e0.elapsed_time(e1)
        n_ph = 1
        cg, cw, co = cmf_step_flops(mpo, mps, cfg.krylov_dim, NSUB_CMF)
        out["mu_cmf_step"] = {"workload": "configs[3] chain, 71 sites, M=128: one second-order CMF step of tau = %g fs (%d RK4 sub-steps per "
                                          "site, Krylov dimension %d at the last site; mean fields built twice per step), one CUDA graph" % (TAU_CMF, NSUB_CMF, cfg.krylov_dim),
                              "ms_per_step": cmf_ms, "steps_timed": n_cmf, "ms_per_fs": cmf_ms / TAU_CMF,
                              "flops": {"gemm": cg, "wstage": cw, "svd_qr": co, "total": cg + cw + co},
                              "frac_fp64_tensor_peak": (products / 4.0 * cg + cw + co) / (cmf_ms * 1e-3) / 1e12 / peak,
                              "launches_per_step": cmf_launches, "norm_sq": nrm, "energy": en,
                              "direct_enqueue_ms": cmf_direct_ms,
                              "phase_ms_per_step": {k: round(v[0] / n_ph, 3) for k, v in ph.items()}}
        out["mu_step"]["ms_per_fs"] = out["mu_step"]["ms_per_step"] / H_MU
        ch.close()
        # configs[4]: the large chain (147 sites, layout B, M = 256): one warm-up and two timed PS steps,
        # gated on invariants (oracle steps at this size take minutes)
        if args.large:
            cfg, mpo, mps = build_chain("fmo256")
            ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim))
            n0, en0 = ch.tdvp_norm_energy()
            ch.tdvp_step_ps(cfg.dt_fs)
            ch.tdvp_sync()
            e0.record()
            for _ in range(2):
                ch.tdvp_step_ps(cfg.dt_fs)
            e1.record()
            ch.tdvp_sync()
            torch.cuda.synchronize()
            nrm, en = ch.tdvp_norm_energy()
            out["ps_step_large"] = {"workload": "configs[4]: FMO-like chain, 7 x 20 modes, layout B, 147 sites, M=256, D_W<=15, "
                                                "k=10, dt=20 fs, CUDA graph",
                                    "ms_per_step": e0.elapsed_time(e1) / 2, "steps_timed": 2, "norm_sq": nrm,
                                    "energy_drift_rel": (en - en0) / abs(en0), "population_sum": float(sum(ch.tdvp_populations(0)))}
            ch.close()
        # the oracle as it stands on the host cores, bounded sample
        v, n, el = time_oracle_heff(M, min_seconds=10.0)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": oracle_cores(), "kind": "oracle",
                               "sample": "%d oracle heff applies (numpy tensordot) of the same M=128 workload in %.1f s" % (n, el)}
    elif rank == 0:
        out["cpu_baseline"] = None
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_ps_only(args):
    """One direct-enqueue (no graph) TDVP-PS step of the configs[3] chain between cudaProfilerStart/Stop,
    after one warm-up step: the target of `ncu --profile-from-start off` for the per-kernel launch list
    of a step (profiles/).  Prints the step's wall time; not a bench value."""
    import torch
    import paper_1907_12044_b200 as T
    cfg, mpo, mps = build_chain("fmo128")
    ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim, flags=T.TDVP_FLAG_NO_GRAPH))
    ch.tdvp_step_ps(cfg.dt_fs)
    ch.tdvp_sync()
    torch.cuda.cudart().cudaProfilerStart()
    t0 = time.perf_counter()
    ch.tdvp_step_ps(cfg.dt_fs)
    ch.tdvp_sync()
    el = time.perf_counter() - t0
    torch.cuda.cudart().cudaProfilerStop()
    print(json.dumps({"ps_step_only_ms": 1e3 * el, "launches": None, "note": "direct enqueue, one step, for profiling"}))
    ch.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the M sweep, the PS step and the CPU baseline")
    ap.add_argument("--large", action="store_true", help="also time the M=256, 147-site chain (about a minute more)")
    ap.add_argument("--ps-step-only", action="store_true", help="one un-graphed TDVP-PS step between cudaProfilerStart/Stop (for ncu)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.ps_step_only:
        run_ps_only(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
