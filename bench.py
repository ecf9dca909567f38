"""bench.py — the CC-LR hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config {1..5}] [--impl ours|reference] [--no-solve]

A "step" is one evaluation of the whole sigma vector  out = (A - (omega + i gamma)) x  (every row of SURVEY.md 8(a)B:
17 terms, layout kernels and the shift) on a batch of nvec trial vectors, through the C ABI (cclr_sigma).  The rows
of 8(a)A (cclr_create) are timed once per run ("create_s"), the rows of 8(a)C-D (cclr_solve + cclr_property) once per
run ("solve": the "time per solve" half of BASELINE.json's metric).  value = algorithmic flops of the packed sigma
(8 real flop per complex multiply-add) of all ranks / max-over-ranks device time.

N > 1 (torchrun): replicas — every rank owns a full context and its own trial vectors (the (operator, frequency)
systems of a response calculation are independent); no data-path collective; "scaling": "weak".

--impl reference times the CPU oracle (oracle/, numpy) on a bounded sample of the workload, rank 0 only.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "CC-LR sigma-vector TFLOP/s (complex FP64)"
UNIT = "TFLOP/s"
ORACLE_SAMPLE = (8, 64)   # (o, v) of the oracle sample: ~7 s per sigma, ~20 s of set-up on 8 host cores


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
def oracle_sigma_timing(steps, warmup):
    """Times oracle.cclr.CCLR.sigma (plain numpy, full tensors) at the sample size with the same input recipe.
    Returns (TFLOP/s with the packed algorithmic flop count, seconds per sigma, cores actually used, sample text)."""
    import synth
    from oracle import ccsd, cclr, packing
    o, v = ORACLE_SAMPLE
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
    sample = ("oracle.cclr.CCLR.sigma (numpy, full unpacked tensors) on the same synthetic recipe at o=%d, v=%d, %d "
              "evaluation(s); the bench workload's full tensors do not fit host memory for the oracle" % (o, v, steps))
    return sigma_flops(o, v) / per / 1e12, per, cores, sample


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    o, v = CONFIGS[args.config]["o"], CONFIGS[args.config]["v"]
    val, per, cores, sample = oracle_sigma_timing(args.steps, min(args.warmup, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": min(args.warmup, 1), "ms_per_step": per * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, o, v), "oracle_sample": "o=%d v=%d" % ORACLE_SAMPLE},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# DRAM traffic of one ladder launch from the ncu captures under profiles/ (bytes; None where no capture exists)
NCU_LADDER_TRAFFIC = {("4m", 3): 7.12e9, ("4m", 4): 43.55e9, ("3m", 3): 7.21e9, ("3m", 4): 48.10e9}

CONFIGS = {1: dict(o=4, v=20, nvec=1), 2: dict(o=10, v=80, nvec=1), 3: dict(o=24, v=200, nvec=1),
           4: dict(o=34, v=300, nvec=1), 5: dict(o=18, v=150, nvec=3)}


def workload_name(cfg, o, v):
    return "BASELINE.json configs[%d]: o=%d v=%d spinors, complex128, packed vvvv (a<b,e<f)" % (cfg - 1, o, v)


# ---------------------------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------------------------
def build_workload(cc, torch, synth, o, v, nvec, seed, ccsd, gemm="3m"):
    """Synthetic inputs generated on the device, context built in place over vvvv."""
    dev = "cuda"
    eri = {k: synth.eri_class(k, o, v, seed=0, device=dev) for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}
    f = synth.fock(o, v, seed=0).to(dev)
    t1, t2 = synth.first_order_amplitudes(o, v, f, eri["oovv"])
    ground = {"kind": "first-order doubles conj<ij||ab>/(e_i+e_j-e_a-e_b), t1=0"}
    if ccsd:   # paper step 1 on the device: converge Omega(t) = 0 to 1e-10 from the first-order guess (cclr_ccsd)
        t1, t2, ginfo = cc.cclr_ccsd(o, v, f, eri, t1, t2, tol=1e-10, maxiter=100)
        ground = {"kind": "cclr_ccsd converged" if ginfo.converged else "cclr_ccsd NOT converged", "iterations": ginfo.iterations,
                  "residual": ginfo.residual, "energy": [ginfo.energy_re, ginfo.energy_im], "seconds": ginfo.seconds}
    torch.cuda.synchronize()
    l0 = cc.cclr_kernel_launches()
    t0 = time.perf_counter()
    ctx = cc.cclr_create(o, v, f, eri, t1, t2, cc.ERI_INPLACE | (cc.GEMM_4M if gemm == "4m" else 0))
    torch.cuda.synchronize()
    create_s = time.perf_counter() - t0
    create_launches = cc.cclr_kernel_launches() - l0
    keep = eri["vvvv"]
    del eri
    x1, x2 = synth.amplitudes(o, v, seed=100 + seed, cls1="x1", cls2="x2", device=dev, nvec=nvec)
    return ctx, keep, x1, x2, create_s, create_launches, ground


def run_ours(args):
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
    ctx, keep, x1, x2, create_s, create_launches, ground = build_workload(cc, torch, synth, o, v, nvec, rank, args.ccsd, args.gemm)
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
                   "gamma": gamma, "sigma_V": synth.sigma_v(v), "ground_state": ground, "parallelism": "replicas x%d" % world,
                   "l2": "inputs larger than L2 (W_vvvv %.2f GB streamed every step)" % (npair(v) ** 2 * 16 / 1e9),
                   "flops_per_step": flops_step, "complex_product": args.gemm, "context_bytes": ctx.bytes()},
        "e2e": {"value": flops_step * world * args.steps / (e2e_ms * 1e-3) / 1e12, "unit": UNIT,
                "h2d_bytes_per_step": (n1 + n2) * nvec * 16, "d2h_bytes_per_step": (n1 + n2) * nvec * 16,
                "ms_per_step": e2e_ms / args.steps},
        "left_sigma": {"ms_per_step": left_ms, "tflops": flops_step / (left_ms * 1e-3) / 1e12},
        "gpu_launches": int(launches), "create_s": create_s, "create_launches": int(create_launches),
    }
    if rank == 0:
        # ---- roofline of the dominant kernel: the pp-ladder DMMA GEMM ---------------------------------------
        peak = cc.cclr_fp64_tensor_peak(20000)
        lad_ms = phases["ladder"] / (args.steps * nvec)
        lad_flops = 8.0 * cm["T11"]
        line["roofline"] = {
            "bound": "tensor", "kernel": "zgemm_kernel<128,%s,16,...,kn,%s> (pp ladder T11)" % ("48" if args.gemm == "3m" else "64", args.gemm),
            "achieved": lad_flops / (lad_ms * 1e-3) / 1e12, "peak": peak, "unit": UNIT,
            "frac": lad_flops / (lad_ms * 1e-3) / 1e12 / peak,
            "complex_product": args.gemm,
            "pipe_frac": (0.75 if args.gemm == "3m" else 1.0) * lad_flops / (lad_ms * 1e-3) / 1e12 / peak,
            "note": "achieved counts 8 real flop per complex multiply-add (SURVEY 8(d) convention, whatever the product); the 3M "
                    "product issues 6 of them on the FP64 tensor pipe (3 real MACs instead of 4), so frac may exceed 1 while "
                    "pipe_frac = executed DMMA flops / peak stays below it",
            "peak_source": "FP64 tensor (DMMA m8n8k4) issue-rate probe cclr_fp64_tensor_peak measured in this run; "
                           "MEASURED_PEAKS.json has no FP64 entry (nominal HGX B200: 37 TFLOP/s)",
            "traffic": NCU_LADDER_TRAFFIC.get((args.gemm, args.config)),
            "traffic_source": "profiles/r01_config4_sigma_step_ncu[_3m].md / r01_zgemm_ncu_full_config3.md "
                              "(dram__bytes_read.sum + dram__bytes_write.sum of the ladder launch)",
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
    # ---- bandwidth kernels against the HBM roofline: the property dot (row D) and the layout kernels of the last sigma step --
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
        line["bandwidth_kernels"] = bw
    # ---- time per solve (rows C, D): 3 right-hand sides x the config's frequencies in one call -----------------
    if not args.no_solve:
        xi1, xi2 = synth.amplitudes(o, v, seed=200 + rank, cls1="x1", cls2="x2", device="cuda", nvec=3)
        omegas = [float(w) for w in torch.linspace(0.05, 0.4, 64)] if args.config == 5 else [0.0, 0.0773]
        barrier()
        t0 = time.perf_counter()
        s1, s2, info = cc.cclr_solve(ctx, xi1, xi2, omegas, gamma, tol=args.tol, maxiter=100)
        prop = cc.cclr_property(ctx, xi1[0].contiguous(), xi2[0].contiguous(), s1[0].contiguous(), s2[0].contiguous())
        torch.cuda.synchronize()
        line["solve"] = {"seconds": time.perf_counter() - t0, "nrhs": 3, "nomega": len(omegas), "gamma": gamma,
                         "tol": args.tol, "iterations": info.iterations, "sigma_calls": info.sigma_calls,
                         "subspace": info.subspace, "converged": info.converged, "max_residual": info.max_residual,
                         "property_abs": abs(prop[0])}
        del s1, s2
    ctx.close()
    if rank == 0:
        if not args.no_cpu:
            val, per, cores, sample = oracle_sigma_timing(2, 0)
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "seconds_per_sigma": per}
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
    ap.add_argument("--ccsd", action="store_true", help="converge the ground-state amplitudes with cclr_ccsd first "
                    "(default: first-order amplitudes; sigma does not depend on the convergence of T, DESIGN.md)")
    ap.add_argument("--gemm", default="3m", choices=["3m", "4m"], help="complex product of the large contractions")
    ap.add_argument("--ops", action="store_true", help="add the per-operation times of the last sigma step to the line")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
