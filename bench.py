"""bench.py — the CC-LR hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config {1..5}] [--impl ours|reference] [--no-solve]

A "step" is one evaluation of the whole sigma vector  out = (A - (omega + i gamma)) x  (every row of SURVEY.md 8(a)B:
17 terms, layout kernels and the shift) on a batch of nvec trial vectors, through the C ABI (cclr_sigma).  value =
algorithmic flops of the packed sigma (8 real flop per complex multiply-add) of all ranks /
max-over-ranks device time.

Timed once per run, on the same context: the paper's workflow — step 1 the ground state (cclr_ccsd, unless
cached or --ground first-order), step 2 the intermediates (cclr_create, "create_s") and the multipliers (cclr_lambda), steps
3-4 the response equations of three synthetic dipole operators at the config's frequencies and the CC-CI response tensor
<<X;Y>> assembled from them (cclr_response_ci_tensor): the "time per solve" half of BASELINE.json's metric.

N > 1 (torchrun): replicas — every rank owns a full context and its own trial vectors (the (operator, frequency)
systems of a response calculation are independent); no data-path collective; "scaling": "weak".

--impl reference times the CPU oracle (oracle/, numpy) on a bounded sample of the workload, rank 0 only.
"""
import argparse
import hashlib
import json
import math
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "CC-LR sigma-vector TFLOP/s (complex FP64)"
UNIT = "TFLOP/s"
ORACLE_SAMPLE = (8, 64)   # (o, v) of the default oracle sample: ~7 s per sigma, ~20 s of set-up on 8 host cores
SPEED_OF_LIGHT_AU = 137.035999084


def npair(n):
    return n * (n - 1) // 2


def sigma_cmacs(o, v):
    """Complex multiply-adds of one packed sigma evaluation, term by term (DESIGN.md table)."""
    oo, vv, ov = npair(o), npair(v), o * v
    t = {
        "S1": v * v * o, "S2": v * o * o, "S3": ov * ov, "S4": ov * ov, "S5": v * o * o * vv, "S6": v * o * v * oo,
        "T1": v * o * v * oo, "T2": vv * o * v * o, "T3": v * v * ov + v * v * v * oo, "T4": o * o * ov + vv * o * o * o,
        "T5": v * v * v * oo, "T6": vv * o * o * o, "T7": vv * oo * oo, "T8": ov * ov * ov,
        "T9": 2 * v * v * v * oo, "T10": 2 * vv * o * o * o, "T11": vv * vv * oo,
    }
    return t


def sigma_flops(o, v):
    return 8.0 * sum(sigma_cmacs(o, v).values())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        load = [s for s, p in zip(sm, pw) if p >= 0.5 * max(pw)] or sm
        load.sort()
        return {"sm_mhz": load[len(load) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------------
# the CPU oracle as it stands, timed on the host cores (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------------------
def oracle_sigma_timing(steps, warmup, sample=None):
    """Times oracle.cclr.CCLR.sigma (plain numpy, full tensors) at the sample size with the same input recipe.
    Returns (TFLOP/s with the packed algorithmic flop count, seconds per sigma, cores actually used, sample text)."""
    import synth
    from oracle import ccsd, cclr, packing
    o, v = sample or ORACLE_SAMPLE
    eri = synth.eri_packed(o, v, seed=0)
    f = synth.fock(o, v)
    t1, t2 = synth.amplitudes(o, v, seed=0, scale=2 * synth.sigma_v(v))
    ints = ccsd.Integrals(o, v, f.numpy(), **packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()}))
    c = cclr.CCLR(ints, *packing.unpack_amplitudes(t1[0].numpy(), t2[0].numpy(), o, v))
    x1, x2 = synth.amplitudes(o, v, seed=3, cls1="x1", cls2="x2")
    X = packing.unpack_amplitudes(x1[0].numpy(), x2[0].numpy(), o, v)
    for _ in range(warmup):
        c.sigma(*X, z=0.0773)
    w0, c0 = time.perf_counter(), time.process_time()
    for _ in range(steps):
        c.sigma(*X, z=0.0773)
    wall, cpu = time.perf_counter() - w0, time.process_time() - c0
    per = wall / steps
    cores = max(1, int(round(cpu / wall)))
    sample_txt = ("oracle.cclr.CCLR.sigma (numpy einsum, full unpacked tensors, as it stands) on the same synthetic recipe at o=%d, "
                  "v=%d, %d evaluation(s); the bench workload's full tensors (v^4 = 130 GB at config 4) do not fit the oracle"
                  % (o, v, steps))
    return sigma_flops(o, v) / per / 1e12, per, cores, sample_txt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    o, v = CONFIGS[args.config]["o"], CONFIGS[args.config]["v"]
    cpu_cfg = getattr(args, "cpu_config", 0)
    sample = (CONFIGS[cpu_cfg]["o"], CONFIGS[cpu_cfg]["v"]) if cpu_cfg else ORACLE_SAMPLE
    val, per, cores, sample_txt = oracle_sigma_timing(args.steps, args.warmup, sample)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": per * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, o, v), "oracle_sample": "o=%d v=%d" % sample, "same_config": False},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_txt, "same_config": False},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


CONFIGS = {1: dict(o=4, v=20, nvec=1), 2: dict(o=10, v=80, nvec=1), 3: dict(o=24, v=200, nvec=1),
           4: dict(o=34, v=300, nvec=1), 5: dict(o=18, v=150, nvec=3)}


def workload_name(cfg, o, v):
    return "BASELINE.json configs[%d]: o=%d v=%d spinors, complex128, packed vvvv (a<b,e<f)" % (cfg - 1, o, v)


def measured_ladder_traffic(gemm, config):
    """DRAM bytes of one ladder launch from an ncu capture of THIS build: profiles/r02_ncu_traffic.csv (rows: sha1 of
    csrc/zgemm.cu, complex product, config, kernel, dram__bytes_read.sum + dram__bytes_write.sum; the command that made it is in
    profiles/r02_ncu_traffic.md).  Returns (bytes, source) or (None, why): the run itself cannot measure DRAM traffic."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_traffic.csv")
    src = os.path.join(ROOT, "paper_2307_14296_b200", "csrc", "zgemm_oz.cu" if gemm == "oz" else "zgemm.cu")
    try:
        with open(src, "rb") as fh:
            sha = hashlib.sha1(fh.read()).hexdigest()
        with open(path) as fh:
            rows = [line.strip().split(",") for line in fh if line.strip() and not line.startswith("#")]
    except OSError:
        return None, "no ncu capture of this build under profiles/"
    for r in rows:
        if len(r) >= 5 and r[0] == sha and r[1] == gemm and r[2] == str(config) and r[3] == "ladder":
            return float(r[4]), "profiles/r02_ncu_traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum of the ladder launch, ncu capture of this build"
    return None, "profiles/r02_ncu_traffic.csv has no capture of this build of csrc/%s for this config / product" % os.path.basename(src)


def measured_peaks():
    """MEASURED_PEAKS.json (driver-written: HBM copy GB/s and cuBLAS bf16 TFLOP/s, burst and sustained) or the profiling guide's
    fallback (6650 GB/s, 1590 burst / 1400 sustained TFLOP/s)."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            p = json.load(fh)
        return {"hbm_gbs": float(p["hbm_gbs"]), "bf16": float(p["bf16_tflops"]), "bf16_sustained": float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                "source": "MEASURED_PEAKS.json (of measured)"}
    except (OSError, KeyError, ValueError):
        return {"hbm_gbs": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0, "source": "B200_PROFILING.md fallback (of fallback)"}


# ---------------------------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------------------------
def ground_state(cc, torch, synth, o, v, f, eri, cfg, mode):
    """Paper step 1.  mode "ccsd": converge Omega(t) = 0 to 1e-10 on the device (cclr_ccsd) from the first-order guess; the
    converged amplitudes are kept in a scratch cache (keyed by config and seed; a cache only skips the recomputation, and the
    cached amplitudes are re-certified by one residual evaluation).  mode "first-order": the perturbative doubles (sigma and
    its timing do not depend on the convergence of T)."""
    t1, t2 = synth.first_order_amplitudes(o, v, f, eri["oovv"])
    if mode != "ccsd":
        return t1, t2, "first-order doubles conj<ij||ab>/(e_i+e_j-e_a-e_b), t1=0 (unconverged)", {}
    cache = os.path.join(os.environ.get("CCLR_CACHE_DIR", os.path.join(tempfile.gettempdir(), "cclr_cache")),
                         "ccsd_cfg%d_seed0_o%d_v%d.pt" % (cfg, o, v))
    if os.path.exists(cache):
        try:
            blob = torch.load(cache, map_location="cuda")
            om1, om2 = cc.cclr_ccsd_residual(o, v, f, eri, blob["t1"], blob["t2"], mode=0)
            res = math.sqrt(float(om1.abs().pow(2).sum()) + 4.0 * float(om2.abs().pow(2).sum()))
            if res <= 1e-9:
                return blob["t1"], blob["t2"], "cclr_ccsd converged (cached; ||Omega|| = %.1e re-evaluated)" % res, blob["info"]
        except Exception:
            pass
    torch.cuda.empty_cache()      # cclr_ccsd sizes its integer-slice operands from the free device memory
    t1, t2, g = cc.cclr_ccsd(o, v, f, eri, t1, t2, tol=1e-10, maxiter=150)
    info = {"iterations": g.iterations, "residual": g.residual, "energy_re": g.energy_re, "energy_im": g.energy_im, "seconds": g.seconds}
    try:
        os.makedirs(os.path.dirname(cache), exist_ok=True)
        torch.save({"t1": t1, "t2": t2, "info": info}, cache)
    except OSError:
        pass
    txt = ("cclr_ccsd converged" if g.converged else "cclr_ccsd NOT converged") + " (%d iterations, %.0f s)" % (g.iterations, g.seconds)
    return t1, t2, txt, info


def build_workload(cc, torch, synth, cfg, o, v, nvec, seed, ground, gemm="3m", graph=True):
    """Synthetic inputs generated on the device, context built in place over vvvv."""
    dev = "cuda"
    eri = {k: synth.eri_class(k, o, v, seed=0, device=dev) for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}
    f = synth.fock(o, v, seed=0).to(dev)
    t1, t2, ground_txt, ground_info = ground_state(cc, torch, synth, o, v, f, eri, cfg, ground)
    torch.cuda.synchronize()
    torch.cuda.empty_cache()      # cclr_create sizes its optional operand copies (sum plane, integer slices) from the free device memory
    l0 = cc.cclr_kernel_launches()
    t0 = time.perf_counter()
    ctx = cc.cclr_create(o, v, f, eri, t1, t2, cc.ERI_INPLACE | (cc.GEMM_4M if gemm == "4m" else 0) | (cc.GEMM_DMMA if gemm == "3m" else 0)
                         | (0 if graph else cc.NO_GRAPH))
    torch.cuda.synchronize()
    create_s = time.perf_counter() - t0
    create_launches = cc.cclr_kernel_launches() - l0
    keep = eri["vvvv"]
    del eri
    torch.cuda.empty_cache()      # hand torch's cached blocks (generator temporaries, the other integral classes) back to the driver: the
                                  # library's solvers size their trial spaces from the free device memory
    x1, x2 = synth.amplitudes(o, v, seed=100 + seed, cls1="x1", cls2="x2", device=dev, nvec=nvec)
    return ctx, keep, x1, x2, create_s, create_launches, ground_txt, ground_info


def time_calls(torch, fn, reps, warm=2):
    """Milliseconds per call on the current stream (CUDA events), after `warm` untimed calls."""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def solver_kernel_bandwidth(cc, torch, ctx, hbm, n, L=24, R=6, nn=6):
    """Rows C3, C5-C7, C9 of SURVEY 8(a)C: the solver's bandwidth kernels alone, at this config's vector length, against the
    measured HBM copy rate.  L = trial vectors, R = systems per multi-row pass, nn = new vectors per iteration (typical sizes of a
    3-component response solve).  Algorithmic bytes: every input element read once, every output element written once."""
    g = torch.Generator(device="cuda")
    g.manual_seed(11)
    rnd = lambda *shape: torch.view_as_complex(torch.randn(*shape, 2, dtype=torch.float64, device="cuda", generator=g))
    V = rnd(2 * L, n)          # [sigma_j ; b_j]
    X = rnd(n)
    Y = torch.empty((R, n), dtype=torch.complex128, device="cuda")
    P = torch.empty((R, n), dtype=torch.complex128, device="cuda")
    coef, z = rnd(R, 2 * L).contiguous(), (rnd(R) * 0.1 + 0.05).contiguous()
    coefL = coef[:, :L].contiguous()
    nrm = torch.empty(R, dtype=torch.float64, device="cuda")
    out = {}

    def rec(name, nbytes, ms, what):
        out[name] = {"bytes": nbytes, "ms": ms, "gbs": nbytes / ms / 1e6, "frac_of_copy_peak": nbytes / ms / 1e6 / hbm, "what": what}

    ms = time_calls(torch, lambda: cc.cclr_vec_block_lincomb(ctx, Y, X, coef, V, nrm2=nrm, z=z, P=P), 5)
    rec("solver residual+norm+precondition (C5+C6 fused)", 16 * n * (2 * L + 1 + 2 * R) + 8 * n, ms,
        "r_k = xi + sum_j beta_kj (sigma_j - z_k b_j), ||r_k||^2 and r_k/(z_k - D) for %d systems over %d subspace vectors, one pass" % (R, 2 * L))
    ms = time_calls(torch, lambda: cc.cclr_vec_block_lincomb(ctx, Y, None, coefL, V[:L]), 5)
    rec("solver solutions t = sum beta b (C9)", 16 * n * (L + R), ms, "%d solutions from %d trial vectors in one pass" % (R, L))
    ms = time_calls(torch, lambda: cc.cclr_vec_block_lincomb(ctx, Y, Y, coefL, V[:L]), 5)
    rec("solver block Gram-Schmidt update V -= b H (C7)", 16 * n * (L + 2 * R), ms, "%d new vectors against %d trial vectors" % (R, L))
    ms = time_calls(torch, lambda: cc.cclr_vec_dots(ctx, V[:L], V[L:L + nn]), 5)
    rec("solver Gram block b^H sigma_new (C3; split-K DMMA GEMM)", 16 * n * (L + nn), ms, "%d x %d sesquilinear dots, every vector read once" % (L, nn))
    ms = time_calls(torch, lambda: cc.cclr_vec_dots(ctx, V[:L], V[L:L + 1]), 5)
    rec("solver projections b^H v (C7; reduction kernel)", 16 * n * (L + 1), ms, "%d dots against one vector" % L)
    del V, X, Y, P
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import synth
    import paper_2307_14296_b200 as cc
    from paper_2307_14296_b200 import replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = CONFIGS[args.config]
    o, v, nvec = cfg["o"], cfg["v"], cfg["nvec"]
    n1, n2 = o * v, npair(o) * npair(v)
    omega, gamma = 0.0773, (0.0045 if args.config in (2, 5) else 0.0)
    ctx, keep, x1, x2, create_s, create_launches, ground_txt, ground_info = build_workload(
        cc, torch, synth, args.config, o, v, nvec, rank, args.ground, args.gemm, not args.no_graph)
    out1, out2 = torch.empty_like(x1), torch.empty_like(x2)
    flops_step = sigma_flops(o, v) * nvec
    cm = sigma_cmacs(o, v)

    # ---- device-resident steps -------------------------------------------------------------------------------
    ctx.set_profiling(True)     # CUDA events between the operations of sigma on the library's stream (phase times)
    for _ in range(args.warmup):
        cc.cclr_sigma(ctx, x1, x2, omega, gamma, out1, out2)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    phases = dict(total=0.0, ladder=0.0, ring=0.0, other_gemm=0.0, layout=0.0)
    launches0 = cc.cclr_kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.nvtx.range_push("timed")     # lets ncu select the timed region: --nvtx --nvtx-include "timed/"
    e0.record()
    for _ in range(args.steps):
        cc.cclr_sigma(ctx, x1, x2, omega, gamma, out1, out2)
        for k, val in ctx.last_sigma_ms().items():
            phases[k] += val
    e1.record()
    torch.cuda.nvtx.range_pop()
    ops_last = ctx.last_sigma_ops()
    barrier()
    launches = cc.cclr_kernel_launches() - launches0
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    ctx.set_profiling(False)

    # ---- the same steps without the per-operation events (the path a solver takes; small configs replay a CUDA graph here) -------
    for _ in range(3):
        cc.cclr_sigma(ctx, x1, x2, omega, gamma, out1, out2)
    barrier()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record()
    for _ in range(args.steps):
        cc.cclr_sigma(ctx, x1, x2, omega, gamma, out1, out2)
    g1.record()
    barrier()
    unprofiled_ms = g0.elapsed_time(g1) / args.steps

    # ---- the same steps with ladder and ring on the FP64 tensor cores (DMMA), same context: the path north_star names -----------
    dmma_ms = None
    if args.gemm == "oz" and ctx.set_gemm_path(0) == 0:
        for _ in range(2):
            cc.cclr_sigma(ctx, x1, x2, omega, gamma, out1, out2)
        barrier()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record()
        for _ in range(3):
            cc.cclr_sigma(ctx, x1, x2, omega, gamma, out1, out2)
        d1.record()
        barrier()
        dmma_ms = d0.elapsed_time(d1) / 3
        oz_on = ctx.set_gemm_path(1) == 1
    else:
        oz_on = False

    # ---- the left transform l (A - z) (Lambda / left response equations; same flop count), 3 steps --------------------------
    for _ in range(2):
        cc.cclr_sigma_left(ctx, x1, x2, omega, gamma, out1, out2)
    barrier()
    l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0.record()
    for _ in range(3):
        cc.cclr_sigma_left(ctx, x1, x2, omega, gamma, out1, out2)
    l1.record()
    barrier()
    left_ms = l0.elapsed_time(l1) / 3

    # ---- end to end: host buffers, copies inside the call ---------------------------------------------------
    hx1, hx2 = x1.cpu().pin_memory(), x2.cpu().pin_memory()
    ho1, ho2 = torch.empty_like(hx1).pin_memory(), torch.empty_like(hx2).pin_memory()
    cc.cclr_sigma_host(ctx, hx1, hx2, omega, gamma, ho1, ho2)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        cc.cclr_sigma_host(ctx, hx1, hx2, omega, gamma, ho1, ho2)   # synchronises before returning
    barrier()
    e2e_s = time.perf_counter() - t0

    ms, e2e_ms = replicas.max_over_ranks([ms, e2e_s * 1e3], device="cuda")
    line = {
        "metric": METRIC, "value": flops_step * world * args.steps / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, o, v), "o": o, "v": v, "nvec": nvec, "omega": omega,
                   "arithmetic": ("complex128 in and out; ladder and ring as integer-slice products on the INT8 tensor path at FP64 accuracy "
                                  "(6 slices of 7 bits, S32 accumulation, FP64 recombination; sigma parity 1e-10 holds, DESIGN.md 6.1b), "
                                  "everything else on the FP64 tensor cores" if oz_on else "complex128 on the FP64 tensor cores (DMMA)"),
                   "gamma": gamma, "sigma_V": synth.sigma_v(v), "ground_state": ground_txt, "parallelism": "replicas x%d" % world,
                   "l2": "inputs larger than L2 (W_vvvv %.2f GB streamed every step)" % (npair(v) ** 2 * 16 / 1e9),
                   "flops_per_step": flops_step, "complex_product": args.gemm, "context_bytes": ctx.bytes()},
        "e2e": {"value": flops_step * world * args.steps / (e2e_ms * 1e-3) / 1e12, "unit": UNIT,
                "h2d_bytes_per_step": (n1 + n2) * nvec * 16, "d2h_bytes_per_step": (n1 + n2) * nvec * 16,
                "ms_per_step": e2e_ms / args.steps},
        "unprofiled": {"ms_per_step": unprofiled_ms, "tflops": flops_step / (unprofiled_ms * 1e-3) / 1e12,
                       "what": "cclr_sigma without the per-operation profiling events%s" % ("" if args.no_graph else " (CUDA-graph replay when the context is small enough)")},
        "left_sigma": {"ms_per_step": left_ms, "tflops": flops_step / (left_ms * 1e-3) / 1e12},
        "integer_slice_path": oz_on,
        "dmma_path": None if dmma_ms is None else {
            "ms_per_step": dmma_ms, "tflops": flops_step / (dmma_ms * 1e-3) / 1e12,
            "what": "the same cclr_sigma on the same context with ladder and ring on the FP64 tensor cores (3M DMMA, cclr_set_gemm_path 0)"},
        "gpu_launches": int(launches), "create_s": create_s, "create_launches": int(create_launches),
        "ground_state_info": ground_info,
    }
    if rank == 0:
        # ---- roofline of the dominant kernel: the pp-ladder DMMA GEMM ---------------------------------------
        peak = cc.cclr_fp64_tensor_peak(20000)
        lad_ms = phases["ladder"] / (args.steps * nvec)
        lad_flops8 = 8.0 * cm["T11"]
        traffic, traffic_src = measured_ladder_traffic(args.gemm, args.config)
        if oz_on:
            # the ladder runs as 21 INT8 slice-pair products (6 slices, t + u <= 5) of the real embedding: 4 real multiply-adds per
            # complex one, 2 ops each -> 21 * 8 vv^2 oo integer ops; peak = measured cuBLAS bf16 (sustained: the kernel is timed inside
            # a long step) x 2, the nominal INT8 : bf16 ratio of the chip (4.5 : 2.25 Pop/s)
            mp = measured_peaks()
            executed = 21.0 * lad_flops8
            peak_i8 = 2.0 * mp["bf16_sustained"]
            line["roofline"] = {
                "bound": "tensor", "kernel": "zgemm_oz_kernel (pp ladder T11 as 21 INT8 slice-pair products, tcgen05.mma.kind::i8, S32 accumulators in TMEM)",
                "achieved": executed / (lad_ms * 1e-3) / 1e12, "peak": peak_i8, "unit": UNIT, "frac": executed / (lad_ms * 1e-3) / 1e12 / peak_i8,
                "flops_counted": "EXECUTED integer ops of the tensor pipe (2 per INT8 multiply-add): 21 slice pairs x 8 vv^2 oo; the duration "
                                 "includes the per-call slicing of the trial vector (the B operand)",
                "peak_source": "2 x bf16_tflops_sustained of %s: the INT8 peak is the bf16 one times the nominal ratio 4.5 : 2.25 "
                               "(burst figure x 2 = %.0f)" % (mp["source"], 2.0 * mp["bf16"]),
                "fp64_equivalent_tflops_8flop_convention": lad_flops8 / (lad_ms * 1e-3) / 1e12,
                "fp64_equivalent_over_dmma_peak": lad_flops8 / (lad_ms * 1e-3) / 1e12 / peak,
                "dmma_peak_measured": peak, "complex_product": "oz (6 integer slices of 7 bits)",
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes": 16.0 * (npair(v) ** 2 + 2 * n2), "ms_per_launch": lad_ms,
            }
        else:
            executed = (0.75 if args.gemm == "3m" else 1.0) * lad_flops8
            line["roofline"] = {
                "bound": "tensor",
                "kernel": "zgemm3m_kernel<48,kn> (pp ladder T11)" if args.gemm == "3m" else "zgemm_kernel<128,64,16,...,kn> (pp ladder T11)",
                "achieved": executed / (lad_ms * 1e-3) / 1e12, "peak": peak, "unit": UNIT,
                "frac": executed / (lad_ms * 1e-3) / 1e12 / peak,
                "flops_counted": "EXECUTED real flops on the FP64 tensor pipe: %d per complex multiply-add of the packed ladder (the 3M "
                                 "product issues 3 real multiply-adds instead of 4); the algorithmic count of SURVEY 8(d), 8 vv^2 oo, is "
                                 "reported beside it" % (6 if args.gemm == "3m" else 8),
                "algorithmic_tflops_8flop_convention": lad_flops8 / (lad_ms * 1e-3) / 1e12,
                "algorithmic_frac_8flop_convention": lad_flops8 / (lad_ms * 1e-3) / 1e12 / peak,
                "complex_product": args.gemm,
                "peak_source": "FP64 tensor (DMMA m8n8k4) issue-rate probe cclr_fp64_tensor_peak measured in this run; "
                               "MEASURED_PEAKS.json has no FP64 entry (nominal HGX B200: 37 TFLOP/s)",
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes": 16.0 * (npair(v) ** 2 + 2 * n2), "ms_per_launch": lad_ms,
            }
        tot = max(phases["total"], 1e-9)
        if args.ops:
            line["ops_ms_last_step"] = [(t, round(m, 4)) for t, m in ops_last]
        line["phases_ms_per_step"] = {k: val / args.steps for k, val in phases.items()}
        line["phase_share"] = {k: val / tot for k, val in phases.items() if k != "total"}
        ring_ms = phases["ring"] / (args.steps * nvec)
        line["ring_tflops"] = 8.0 * cm["T8"] / (ring_ms * 1e-3) / 1e12
        line["fp64_pipe_probe_tflops"] = {"dmma": peak, "dfma": cc.cclr_fp64_pipe_probe(1), "dmma+dfma by warp": cc.cclr_fp64_pipe_probe(2)}
        line["hbm_copy_gbs_measured"] = cc.cclr_hbm_copy_peak(4 << 30)
        line["clocks"] = clocks
    # ---- bandwidth kernels against the HBM roofline: property dot (row D), layout kernels of the last sigma step, solver kernels --
    reps = 20
    cc.cclr_property(ctx, x1[0].contiguous(), x2[0].contiguous(), out1[:1].contiguous(), out2[:1].contiguous())
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(reps):
        cc.cclr_property(ctx, x1[0], x2[0], out1[:1], out2[:1])       # synchronises: returns host data
    dot_s = (time.perf_counter() - t0) / reps
    if rank == 0:
        hbm = line["hbm_copy_gbs_measured"]
        oo, vv = npair(o), npair(v)
        layout_bytes = {   # algorithmic bytes: every source element read once, every destination element written once
            "perm Ur[ea(ij)]": 16 * (n2 + v * v * oo), "perm Xt[im(ef)]": 16 * (n2 + o * o * vv),
            "perm R[aiem]": 16 * (n2 + (o * v) ** 2), "perm Xo[(ab)in]": 16 * (n2 + vv * o * o),
            "perm out2[(ab)(ij)]": 16 * (3 * n2 + v * v * oo + vv * o * o + (o * v) ** 2),
        }
        bw = {"property_dot": {"bytes": 32 * (n1 + n2), "ms": dot_s * 1e3, "gbs": 32 * (n1 + n2) / dot_s / 1e9,
                               "frac_of_copy_peak": 32 * (n1 + n2) / dot_s / 1e9 / hbm}}
        for text, msv in ops_last:
            for key, nbytes in layout_bytes.items():
                if text.startswith(key) and msv > 0:
                    per = msv / nvec
                    bw[key] = {"bytes": nbytes, "ms": per, "gbs": nbytes / per / 1e6, "frac_of_copy_peak": nbytes / per / 1e6 / hbm}
        bw.update(solver_kernel_bandwidth(cc, torch, ctx, hbm, n1 + n2))
        line["bandwidth_kernels"] = bw
    # ---- time per solve: paper steps 2-4 for three dipole operators at the config's frequencies -----------------------
    if not args.no_solve:
        nop = 4 if args.config == 3 else 3     # config 3 adds the imaginary-antisymmetric operator (optical-rotation pair, Eq. 36)
        ops = [synth.hermitian_operator(o + v, 0, c) for c in range(3)]
        if nop == 4:
            ops.append(synth.hermitian_operator(o + v, 0, 3, imaginary_antisymmetric=True))
        X = torch.from_numpy(np.stack(ops)).cuda().contiguous()
        omegas = [float(w) for w in np.linspace(0.05, 0.4, 64)] if args.config == 5 else [0.0, 0.0773]
        barrier()
        torch.cuda.empty_cache()
        free_b, total_b = torch.cuda.mem_get_info()
        t0 = time.perf_counter()
        lam1, lam2, linfo = cc.cclr_lambda(ctx, tol=args.tol, maxiter=200)
        torch.cuda.synchronize()
        lam_s = time.perf_counter() - t0
        t0 = time.perf_counter()
        tensor, info = cc.cclr_response_ci_tensor(ctx, X, omegas, gamma, tol=args.tol, maxiter=200)
        torch.cuda.synchronize()
        resp_s = time.perf_counter() - t0
        nshift = len(set(omegas) | set(-w for w in omegas))
        nsys = nop * nshift * (2 if gamma != 0.0 else 1)
        sol = {"what": "cclr_lambda, then cclr_response_ci_tensor: xi / EOM-eta of %d operators, %d response systems (A - z) t = -xi "
                       "(shifts +-omega%s) in shared trial spaces, CC-CI <<X;Y>>_omega for every pair (Eq. 16-17)"
                       % (nop, nsys, ", both signs of gamma" if gamma != 0.0 else ""),
               "seconds": lam_s + resp_s, "lambda_seconds": lam_s, "lambda_sigma_calls": linfo.sigma_calls, "lambda_converged": linfo.converged,
               "response_seconds": resp_s, "response_sigma_calls": info.sigma_calls, "response_iterations": info.iterations,
               "subspace": info.subspace, "converged": info.converged, "max_residual": info.max_residual, "systems": nsys,
               "seconds_per_system": resp_s / nsys, "free_device_gb_before": free_b / 1e9, "nop": nop, "nomega": len(omegas), "gamma": gamma, "tol": args.tol}
        show = [0, len(omegas) - 1] if len(omegas) > 2 else list(range(len(omegas)))
        sol["alpha_xx_yy_zz"] = {"%.4f" % omegas[k]: [[-tensor[k][r][r].real, -tensor[k][r][r].imag] for r in range(3)] for k in show}
        sol["alpha_xy"] = {"%.4f" % omegas[k]: [-tensor[k][0][1].real, -tensor[k][0][1].imag] for k in show}
        if nop == 4:
            sol["optical_rotation_Gprime_x (-Im<<mu_x;m>>)"] = {"%.4f" % omegas[k]: -tensor[k][0][3].imag for k in show}
        if gamma != 0.0:   # sigma_abs(omega) = 4 pi omega / c * Im mean alpha (Eq. 22)
            sol["sigma_abs"] = [4.0 * math.pi * w / SPEED_OF_LIGHT_AU * sum(-tensor[k][r][r].imag for r in range(3)) / 3.0
                                for k, w in enumerate(omegas)]
        line["solve"] = sol
    ctx.close()
    if rank == 0:
        if not args.no_cpu:
            sample = (CONFIGS[args.cpu_config]["o"], CONFIGS[args.cpu_config]["v"]) if args.cpu_config else ORACLE_SAMPLE
            val, per, cores, sample_txt = oracle_sigma_timing(1 if args.cpu_config else 2, 0, sample)
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_txt,
                                    "seconds_per_sigma": per, "same_config": sample == (o, v)}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--no-solve", action="store_true")
    ap.add_argument("--ground", default="ccsd", choices=["ccsd", "first-order"],
                    help="ground-state amplitudes: converged on the device with cclr_ccsd (default; cached in a scratch directory) "
                         "or the first-order doubles (sigma does not depend on the convergence of T, DESIGN.md)")
    ap.add_argument("--gemm", default="oz", choices=["3m", "4m", "oz"],
                    help="complex product of the large contractions: 3M / 4M on the FP64 tensor cores (DMMA), or oz = ladder and ring as "
                         "integer-slice products on the INT8 tensor path at FP64 accuracy (the library default; 3m / 4m set CCLR_GEMM_DMMA / CCLR_GEMM_4M)")
    ap.add_argument("--no-graph", action="store_true", help="do not replay sigma as a CUDA graph (small configs; before / after numbers)")
    ap.add_argument("--ops", action="store_true", help="add the per-operation times of the last sigma step to the line")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--cpu-config", type=int, default=0, choices=[0, 1, 2], help="time the oracle at this BASELINE config instead of "
                    "the default o=8, v=64 sample (config 2: ~1.5 min of set-up and 20 s per sigma on 8 cores)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
