#!/usr/bin/env python
"""Benchmark of the THC-RR-CCSD projected doubles residual + energy on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

One "step" = one pass of the whole hot path: thc_residual (R_PQ, all six terms)
followed by thc_energy_device, on one seeded synthetic input set of BASELINE.json config C (default 1).
Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for how every field is measured.

--impl reference times the CPU oracle (oracle/dense.py) as it stands on the host cores; this and the
`cpu_baseline` leg are the only places that execute anything under oracle/.
"""
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

METRIC = "thc_ccsd_residual_evals_per_sec"
UNIT = "evals/s"
INPUT_NAMES = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")

# Nominal figures used for the FP64 roofline denominators:
#   FP64 tensor (DMMA): MEASURED_PEAKS.json bf16_tflops x (nominal FP64 tensor 45 / nominal bf16 2250), the ratio
#   of /opt/skills/guides/blackwell_cuda_programming.md's table;  FP64 FMA pipe: 148 SMs x 64 DFMA lanes x 2 flop
#   x SM clock.
NOMINAL_FP64_TENSOR_OVER_BF16 = 45.0 / 2250.0
SMS, DFMA_LANES_PER_SM = 148, 64
FALLBACK_BF16_TFLOPS, FALLBACK_HBM_GBS, FALLBACK_SM_MAX_MHZ = 1590.0, 6650.0, 1965.0

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed `ncu --set full`
# capture (profiles/), keyed by (config, kernel class); None until captured.  For a class of many launches (gemm) it is
# the class's DRAM bytes of one evaluation / its launches per evaluation.  Source: profiles/r01_dram_traffic.md.
NCU_TRAFFIC_BYTES = {(1, "gemm"): 93.26e6, (2, "triple"): 804.5e9}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    hbm=d["hbm_gbs"], sm_max_mhz=d.get("sm_max_mhz", FALLBACK_SM_MAX_MHZ), source="measured")
    return dict(bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=1400.0, hbm=FALLBACK_HBM_GBS,
                sm_max_mhz=FALLBACK_SM_MAX_MHZ, source="fallback")


def dense_oracle_flops(o, v, NL):
    """Rough flop count of the dense oracle: ERI builds + the Omega contractions."""
    return 2.0 * (o ** 2 * v ** 4 + o ** 4 * v ** 2 + 6 * o ** 3 * v ** 3) + 2.0 * NL * v ** 4


def time_oracle(cfg, reps, budget_s=30.0):
    """Time oracle/dense.py on config `cfg` if its dense arrays fit (configs 0, 1); for larger configs time
    config 1 and scale by the dense-oracle flop ratio (stated in `sample`)."""
    import numpy as np
    from thc_synth import make_config, config_dims
    from oracle import dense
    run_cfg = cfg if cfg <= 1 else 1
    x = make_config(run_cfg)
    times = []
    t_all = time.perf_counter()
    for _ in range(max(1, reps)):
        t0 = time.perf_counter()
        res = dense.residual_and_energy(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
        times.append(time.perf_counter() - t0)
        assert np.isfinite(res["R"]).all()
        if time.perf_counter() - t_all > budget_s:
            break
    t = statistics.median(times)
    cores = len(os.sched_getaffinity(0))
    if run_cfg == cfg:
        value, sample = 1.0 / t, f"{len(times)} full dense-oracle evaluation(s) of config {cfg} (median)"
    else:
        o, v, NL, _, _ = config_dims(cfg)
        o1, v1, NL1, _, _ = config_dims(1)
        scale = dense_oracle_flops(o, v, NL) / dense_oracle_flops(o1, v1, NL1)
        value = 1.0 / (t * scale)
        sample = (f"{len(times)} full dense-oracle evaluation(s) of config 1, extrapolated to config {cfg} by the "
                  f"dense-oracle flop ratio {scale:.3g} (its dense t/ERI arrays do not fit host memory at config {cfg})")
    return dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample, seconds_per_eval=1.0 / value)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from thc_synth import config_dims
    o, v, NL, NP, NX = config_dims(args.config)
    n = args.steps + args.warmup
    per_eval_budget = 150.0 / max(1, n)
    import numpy as np
    from thc_synth import make_config
    from oracle import dense
    run_cfg = args.config if args.config <= 1 else 1
    x = make_config(run_cfg)

    def step():
        res = dense.residual_and_energy(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
        assert np.isfinite(res["R"]).all()

    # each step is one full dense-oracle evaluation unless that would take the run past a few minutes; then a
    # step is the oracle on config 0 scaled by the flop ratio (bounded sample)
    t0 = time.perf_counter(); step(); first = time.perf_counter() - t0
    sample_cfg = run_cfg
    if first > per_eval_budget and run_cfg != 0:
        sample_cfg = 0
        x = make_config(0)
    for _ in range(max(0, args.warmup - 1)):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    so, sv, sNL, _, _ = config_dims(sample_cfg)
    scale = dense_oracle_flops(o, v, NL) / dense_oracle_flops(so, sv, sNL)
    value = 1.0 / (dt * scale)
    cores = len(os.sched_getaffinity(0))
    sample = (f"each step = one full dense-oracle evaluation of config {sample_cfg}" +
              ("" if sample_cfg == args.config else f", extrapolated to config {args.config} by flop ratio {scale:.3g}"))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * scale * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config{args.config}", "o": o, "v": v, "NL": NL, "NP": NP, "NX": NX},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.proc, self.idx = None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in out.strip().splitlines():
            f = [s.strip() for s in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for nm, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2111_11473_b200 as thc
    from thc_synth import make_inputs, CONFIGS

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the THC residual has no CPU path)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    thc.lib()      # fails loudly if the extension is missing

    c = CONFIGS[args.config]
    o, v, NL, NP, NX = c["o"], c["v"], c["NL"], c["NP"], c["NX"]
    # N = 1: the whole evaluation on one GPU.  N > 1: ONE evaluation sharded over the ranks as the paper shards it
    # (Cholesky ranges + row blocks of the T2^2 terms, one NCCL all-reduce) -> strong scaling.
    sharded = world > 1 or bool(os.environ.get("THC_BENCH_FORCE_SHARDED"))    # the env switch exercises the sharded code path on one rank
    L0, L1, _, _ = thc.thc_shard_range(NL, NP, rank, world)
    provider = args.config >= 4                      # B_vv (304 GB) is generated block by block on the device
    if args.config <= 2:
        x = make_inputs(o, v, NL, NP, NX, seed=c["seed"])
        host = [torch.from_numpy(np.ascontiguousarray(getattr(x, n))).pin_memory() for n in INPUT_NAMES]
        if sharded:
            for k in (3, 4, 5):
                host[k] = host[k][L0:L1].contiguous().pin_memory()
        d = [t.to(dev, non_blocking=True) for t in host]
    else:
        from thc_synth import device as synth
        dd = synth.make_inputs_device(o, v, NL, NP, NX, c["seed"], device=dev, with_bvv=False)
        if sharded:
            dd["B_ov"], dd["B_oo"] = dd["B_ov"][L0:L1].contiguous(), dd["B_oo"][L0:L1].contiguous()
        if not provider:
            dd["B_vv"] = synth.bvv_block(c["seed"], o, v, NL, L0, L1, dev)
        d = [dd[nm] for nm in INPUT_NAMES]
        host = [None if t is None else t.cpu().pin_memory() for t in d]
    if provider:
        from thc_synth import device as synth

        def bvv_fill(Lg, nl, dst):                   # thc_bvv_provider: fills B_vv[Lg:Lg+nl] on the library's stream
            synth.bvv_block(c["seed"], o, v, NL, Lg, Lg + nl, dev, out=dst)
        d[5] = bvv_fill
        host[5] = bvv_fill
    R = torch.empty(NP, NP, dtype=torch.float64, device=dev)
    E = torch.zeros(1, dtype=torch.float64, device=dev)
    R_host = torch.empty(NP, NP, dtype=torch.float64).pin_memory()
    h = thc.thc_setup(o, v, NL, NP, NX, bvv_mode="provider" if provider else "device")
    flops = h.algorithmic_flops
    input_bytes = sum(t.numel() * 8 for t in host if torch.is_tensor(t))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    use_flush = input_bytes < (512 << 20)
    if sharded:
        from paper_2111_11473_b200.sharded import CudaBackend, residual_sharded, energy_sharded
        backend = CudaBackend(h, *d)

    def step():
        if sharded:
            R.copy_(residual_sharded(backend))
            E.copy_(energy_sharded(backend))
        else:
            h.thc_residual(*d, out=R)
            h.thc_energy_device(d[0], d[1], d[2], d[3], out=E)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- warm-up (also finds the dominant kernel class) ----
    W = max(3, args.warmup)
    for _ in range(W - 1):
        step()
    h.thc_profile_begin(7)
    step()
    prof_w = h.thc_profile_end()
    work_w = h.thc_profile_work()        # executed flop (gemm, triple) / algorithmic HBM bytes (ew) of that step
    dominant = max(prof_w, key=lambda k: prof_w[k][0])
    dom_bit = {"gemm": 1, "triple": 2, "ew": 4}[dominant]

    # ---- timed region: K steps, device-timed, L2 flushed between steps ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    K = args.steps
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    launches0 = h.kernel_launches
    barrier()
    wall0 = time.perf_counter()
    h.thc_profile_begin(dom_bit)
    for k in range(K):
        if use_flush:
            flush.fill_(k & 0xFF)
        ev[k][0].record()
        step()
        ev[k][1].record()
    prof = h.thc_profile_end()           # synchronises the stream
    barrier()
    wall = time.perf_counter() - wall0
    launches = h.kernel_launches - launches0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_s = float(total_ms.item()) * 1e-3
    value = (1 if sharded else world) * K / total_s
    E_val = float(E.item())

    # ---- end to end through thc_residual_host: pinned host buffers in, R + E back on the host, every step ----
    # (N > 1: the sharded evaluation has no host-buffer entry; its inputs are copied H2D explicitly every step)
    def e2e_step():
        if sharded:
            dh = [t.to(dev, non_blocking=True) if torch.is_tensor(t) else t for t in host]
            be = CudaBackend(h, *dh)
            R_host.copy_(residual_sharded(be), non_blocking=True)
            Eh = energy_sharded(be).cpu()
            torch.cuda.synchronize()
            return float(Eh[0])
        return h.thc_residual_host(*host, R_host)       # synchronous

    Ke = max(1, min(K, 5 if args.config == 2 else (1 if args.config >= 3 else K)))
    if args.config >= 4:
        # config 4: staging copies of the 38 GB of resident inputs do not fit beside them and the workspace
        Ke, e2e_value = 0, None
    else:
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            e2e_step()
        barrier()
        e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
        e2e_value = (1 if sharded else world) * Ke / float(e2e_s.item())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class ----
    pk = measured_peaks()
    dom_ms, dom_n = prof[dominant]
    per_eval_ms = dom_ms / K
    fo, fv, fNL, fNP, fNX = float(o), float(v), float(NL), float(NP), float(NX)
    triple_flops = 5.0 * fNX * fNP ** 3
    ew_flops = 5.0 * fNL * fNP * fNP
    if dominant == "triple":
        alg = triple_flops
        peak = SMS * DFMA_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
        roof = {"bound": "alu", "kernel": "triple_product_kernel (Alg.6 line 11)", "achieved": alg / (per_eval_ms * 1e-3) / 1e12,
                "peak": peak, "unit": "TFLOP/s",
                "peak_source": f"148 SMs x 64 FP64 FMA lanes x 2 flop x {pk['sm_max_mhz']:.0f} MHz (max SM clock, {pk['source']})"}
    elif dominant == "gemm":
        alg = flops - triple_flops - ew_flops
        peak = pk["bf16"] * NOMINAL_FP64_TENSOR_OVER_BF16
        roof = {"bound": "tensor", "kernel": "dgemm_kernel (FP64 DMMA, all GEMM chains)", "achieved": alg / (per_eval_ms * 1e-3) / 1e12,
                "peak": peak, "unit": "TFLOP/s",
                "peak_source": f"{pk['source']} bf16 {pk['bf16']:.1f} TFLOP/s x nominal FP64-tensor/bf16 ratio 45/2250"}
    else:
        alg = 0.0
        roof = {"bound": "hbm", "kernel": "Hadamard/reduction kernels", "achieved": None, "peak": pk["hbm"], "unit": "GB/s",
                "peak_source": f"{pk['source']} copy bandwidth"}
    if roof["achieved"] is not None:
        roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"] = NCU_TRAFFIC_BYTES.get((args.config, dominant))
    roof["launches_per_step"] = dom_n / K
    roof["ms_per_step"] = per_eval_ms
    roof["share_of_step"] = per_eval_ms / (1e3 * total_s / K)
    roof["class_ms_warmup_step"] = {k: round(prof_w[k][0], 4) for k in prof_w}
    # every kernel class of one profiled warm-up step against its own roof (EXECUTED work, recomputation included)
    dmma_probe = SMS * DFMA_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    per_class = {}
    for k, (unit, peak, bound) in {"gemm": ("TFLOP/s", pk["bf16"] * NOMINAL_FP64_TENSOR_OVER_BF16, "tensor"),
                                   "triple": ("TFLOP/s", dmma_probe, "alu"),
                                   "ew": ("GB/s", pk["hbm"], "hbm")}.items():
        ms_k = prof_w[k][0]
        if ms_k <= 0:
            continue
        ach = work_w[k] / (ms_k * 1e-3) / (1e12 if unit == "TFLOP/s" else 1e9)
        per_class[k] = {"bound": bound, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
                        "ms": round(ms_k, 4), "launches": prof_w[k][1]}
    per_class["gemm"]["frac_of_dmma_issue_rate"] = per_class["gemm"]["achieved"] / dmma_probe if "gemm" in per_class else None

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": 1e3 * total_s / K, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config{args.config}", "o": o, "v": v, "NL": NL, "NP": NP, "NX": NX, "seed": c["seed"],
                       "blocks": h.blocks, "l2": "flushed between steps (256 MiB write)" if use_flush else "inputs larger than L2",
                       "parallelism": "1 GPU" if world == 1 else f"one evaluation sharded over {world} GPUs (Cholesky ranges + T2^2 row blocks, one all-reduce)",
                       "B_vv": "provider callback, generated per L-block on the device" if provider else "resident in HBM"},
            "tflops_fp64_algorithmic": (1 if sharded else world) * flops * K / total_s / 1e12,
            "algorithmic_flops_per_eval": flops, "energy_Eh": E_val,
            "wall_s_timed_region": wall, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": input_bytes, "d2h_bytes_per_step": NP * NP * 8 + 8,
                    "steps": Ke},
            "gpu_launches": launches, "roofline": roof, "rooflines_by_class": per_class}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(args.config, reps=3)
    print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
