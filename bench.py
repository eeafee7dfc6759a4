#!/usr/bin/env python
"""Benchmark of the THC-RR-CCSD projected doubles residual + energy on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]
                    [--bvv device|host|provider] [--trace FILE] [--probe] [--no-cpu-baseline]
                    [--workload residual|second]

One "step" = one pass of the whole hot path: thc_residual (R_PQ, all six terms)
followed by thc_energy_device, on one seeded synthetic input set of BASELINE.json config C.  The default workload is
config 3 (o=150, v=850, NL=3000, NP=2500, NX=5000), the largest configuration whose 25 evaluations fit the driver's
bench window; config 4 takes ~13 minutes per evaluation and is benched with --config 4.
Prints ONE JSON line (rank 0).  DESIGN.md section 8 says how every field is measured.

--impl reference times the CPU oracle (oracle/) as it stands on the host cores; this and the `cpu_baseline` leg are
the only places that execute anything under oracle/.  --probe prints the measured FP64 / shared-memory ceilings of
the device (the denominators DESIGN.md section 7 discusses) instead of running the benchmark.
"""
import argparse
import csv
import json
import os
import socket
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
#   x SM clock.  The same-run yardsticks (`extra.yardstick`) show what the pipe really delivers.
NOMINAL_FP64_TENSOR_OVER_BF16 = 45.0 / 2250.0
SMS, DFMA_LANES_PER_SM = 148, 64
FALLBACK_BF16_TFLOPS, FALLBACK_HBM_GBS, FALLBACK_SM_MAX_MHZ = 1590.0, 6650.0, 1965.0
# DRAM bytes per launch of a kernel class from a committed `ncu --set full` capture: profiles/<this file>, one row per
# (config, class) with the command that produced it.  No row -> roofline.traffic is null.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    hbm=d["hbm_gbs"], sm_max_mhz=d.get("sm_max_mhz", FALLBACK_SM_MAX_MHZ), source="measured")
    return dict(bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=1400.0, hbm=FALLBACK_HBM_GBS,
                sm_max_mhz=FALLBACK_SM_MAX_MHZ, source="fallback")


def ncu_traffic(config, cls):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu summary, or None."""
    if not os.path.exists(TRAFFIC_CSV):
        return None
    with open(TRAFFIC_CSV) as f:
        for row in csv.DictReader(f):
            if int(row["config"]) == config and row["class"] == cls:
                return float(row["dram_bytes_per_launch"])
    return None


# ======================================================================================================================
# CPU oracle legs (cpu_baseline and --impl reference)
# ======================================================================================================================
def dense_oracle_flops(o, v, NL):
    """Rough flop count of the dense oracle: ERI builds + the Omega contractions."""
    return 2.0 * (o ** 2 * v ** 4 + o ** 4 * v ** 2 + 6 * o ** 3 * v ** 3) + 2.0 * NL * v ** 4


class OracleSample:
    """A bounded sample of one oracle evaluation of config `cfg`, and the factor that scales its time to a whole one.

    configs 0, 1: the dense oracle (oracle/dense.py), the whole evaluation (scale 1).
    configs 2-4 : the dense arrays do not fit host memory, so the oracle of record there is the sampled-row oracle
                  (oracle/rows.py).  The sample is one row R[P, :] of all six terms over the FIRST `nl` Cholesky vectors
                  (+ the xi intermediates and the energy over the same vectors); a whole evaluation is NP rows, and the
                  Cholesky-dependent work (sigma1, sigma2, sigma3, xi, E) grows by NL / nl.  The sigma6 row, which alone
                  takes minutes at config 3, is a sum over the ERI grid points I of identical pieces (THC ERIs expanded
                  over (I, J), J always the whole grid): the sample evaluates it for the FIRST `nxi` points I (the oracle
                  is handed the first nxi rows of V) and its time grows by NX / nxi.  All three factors are stated in
                  `sample`; a step is a few seconds of CPU work.
    """

    def __init__(self, cfg, nl=None):
        from thc_synth import CONFIGS, make_inputs
        c = CONFIGS[cfg]
        self.cfg, self.c = cfg, c
        if cfg <= 1:
            self.x = make_inputs(c["o"], c["v"], c["NL"], c["NP"], c["NX"], c["seed"])
            self.kind = "dense"
            self.sample = f"one full dense-oracle evaluation of config {cfg}"
        else:
            self.nl = nl or {2: 8, 3: 2, 4: 1}[cfg]
            self.nxi = {2: 256, 3: 64, 4: 16}[cfg]
            self.x = make_inputs(c["o"], c["v"], c["NL"], c["NP"], c["NX"], c["seed"], l_keep=self.nl)
            self.kind = "rows"
            self.P = c["NP"] // 2
            self.sample = (f"sampled-row oracle (oracle/rows.py) on config {cfg}: one row P={self.P} of sigma1..sigma9, xi and E "
                           f"over the first {self.nl} of {c['NL']} Cholesky vectors, the sigma6 row over the first {self.nxi} of "
                           f"{c['NX']} outer ERI-grid points; a whole evaluation = NP={c['NP']} rows, Cholesky-dependent parts "
                           f"x{c['NL'] / self.nl:.0f}, sigma6 x{c['NX'] / self.nxi:.1f}")

    def run(self):
        """Returns the estimated seconds of ONE whole oracle evaluation of the config; self.last_wall_s = what the
        sample itself took."""
        t_wall = time.perf_counter()
        est = self._run()
        self.last_wall_s = time.perf_counter() - t_wall
        return est

    def _run(self):
        import numpy as np
        x = self.x
        if self.kind == "dense":
            from oracle import dense
            t0 = time.perf_counter()
            res = dense.residual_and_energy(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
            dt = time.perf_counter() - t0
            assert np.isfinite(res["R"]).all()
            return dt
        from oracle.rows import RowOracle
        ro = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps, lblock=self.nl)
        c, lscale = self.c, self.c["NL"] / self.nl
        t0 = time.perf_counter()
        ro.xi(); ro.energy()
        t_once = (time.perf_counter() - t0) * lscale                       # once per evaluation, all L
        t0 = time.perf_counter()
        r = ro.row(self.P, terms=("s1", "s2", "s3"))
        t_lin = (time.perf_counter() - t0) * lscale                        # per row, all L
        t0 = time.perf_counter()
        r.update(ro.row(self.P, terms=("s7", "s9")))
        t_quad = time.perf_counter() - t0                                  # per row, no L dependence
        ro6 = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V[: self.nxi], x.eps, lblock=self.nl)
        t0 = time.perf_counter()
        r.update(ro6.row(self.P, terms=("s6",)))                           # outer grid points I < nxi only
        t_s6 = (time.perf_counter() - t0) * c["NX"] / self.nxi
        assert all(np.isfinite(v).all() for v in r.values())
        return t_once + c["NP"] * (t_lin + t_quad + t_s6)


def time_oracle(cfg, budget_s=30.0):
    cores = len(os.sched_getaffinity(0))
    s = OracleSample(cfg)
    times, t_all = [], time.perf_counter()
    while len(times) < 3 and (not times or time.perf_counter() - t_all < budget_s):
        times.append(s.run())
    t = statistics.median(times)
    return dict(value=1.0 / t, unit=UNIT, cores=cores, kind="oracle", sample=f"{s.sample}; median of {len(times)} run(s)",
                seconds_per_eval=t)


def run_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from thc_synth import config_dims
    o, v, NL, NP, NX = config_dims(args.config)
    s = OracleSample(args.config)
    for _ in range(args.warmup):
        s.run()
    times, walls = [], []
    for _ in range(args.steps):
        times.append(s.run())
        walls.append(s.last_wall_s)
    dt = sum(times) / len(times)                     # seconds of one WHOLE evaluation (the sample's time scaled up)
    cores = len(os.sched_getaffinity(0))
    value = 1.0 / dt
    # ms_per_step is what a step (= one bounded sample) really took, so that steps x ms_per_step is this run's timed region;
    # `value` is whole evaluations per second, i.e. 1 / seconds_per_eval_extrapolated
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(walls) / len(walls), "seconds_per_eval_extrapolated": dt,
            "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config{args.config}", "o": o, "v": v, "NL": NL, "NP": NP, "NX": NX},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"each step = {s.sample}"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ======================================================================================================================
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
                                          "--format=csv,noheader,nounits", "-lms", "200"],
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


def yardstick(thc, torch, dev, n=8192):
    """FP64 GEMM n^3 through the library's own DMMA kernel (thc_dgemm) and through torch.matmul (cuBLAS), best of 3
    after one warm-up, TFLOP/s each: what the FP64 tensor pipe delivers in this very run.  cuBLAS is
    a yardstick only, never on the product path."""
    out = {}
    try:
        g = torch.Generator(device=dev).manual_seed(7)
        A = torch.randn(n, n, dtype=torch.float64, device=dev, generator=g)
        B = torch.randn(n, n, dtype=torch.float64, device=dev, generator=g)
        C = torch.empty(n, n, dtype=torch.float64, device=dev)
        hy = thc.thc_setup(4, 8, 4, 16, 16)

        def best(fn):
            fn()
            ts = []
            for _ in range(3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record(); b.synchronize()
                ts.append(a.elapsed_time(b))
            return 2.0 * n ** 3 / (min(ts) * 1e-3) / 1e12
        out["thc_dgemm_8192_tflops"] = best(lambda: hy.thc_dgemm(1, 1, n, n, n, 1.0, A, n, B, n, 0.0, C, n))
        out["torch_matmul_fp64_8192_tflops"] = best(lambda: torch.matmul(A, B.T, out=C))
        hy.close()
        del A, B, C
        torch.cuda.empty_cache()
    except Exception as exc:          # the yardstick must never take the benchmark down (e.g. memory at config 4)
        out["error"] = repr(exc)
    return out


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` (N > 1) without a launcher: start N ranks, one per GPU, through torch.distributed.run.
    Fails loudly when the node has fewer GPUs -- never a silent N = 1 run."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} requested but this node has {have} CUDA device(s)")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")            # the communicator lines show the ranks / NVLS in the log
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd, env=env))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2111_11473_b200 as thc
    from thc_synth import make_inputs, CONFIGS

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the THC residual has no CPU path)")
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit(f"bench.py: rank {rank} has no GPU (LOCAL_RANK {local_rank}, {torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        dist.init_process_group("nccl", device_id=dev)
    thc.lib()      # fails loudly if the extension is missing

    c = CONFIGS[args.config]
    o, v, NL, NP, NX = c["o"], c["v"], c["NL"], c["NP"], c["NX"]
    # N = 1: the whole evaluation on one GPU.  N > 1: ONE evaluation sharded over the ranks as the paper shards it
    # (Cholesky ranges + row blocks of the T2^2 terms, one NCCL all-reduce) -> strong scaling.
    sharded = world > 1
    L0, L1, _, _ = thc.thc_shard_range(NL, NP, rank, world)
    bvv_mode = args.bvv or ("provider" if args.config >= 4 else "device")
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
        if bvv_mode != "provider":
            dd["B_vv"] = synth.bvv_block(c["seed"], o, v, NL, L0, L1, dev)
        d = [dd[nm] for nm in INPUT_NAMES]
        host = [None if t is None else t.cpu().pin_memory() for t in d]
        del dd
    if bvv_mode == "provider":
        from thc_synth import device as synth

        def bvv_fill(Lg, nl, dst):                   # thc_bvv_provider: fills B_vv[Lg:Lg+nl] on the library's stream
            synth.bvv_block(c["seed"], o, v, NL, Lg, Lg + nl, dev, out=dst)
        d[5] = bvv_fill
        host[5] = bvv_fill
    elif bvv_mode == "host":                         # B_vv stays in pinned host memory and is streamed per L-block
        d[5] = host[5]
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    R = torch.empty(NP, NP, dtype=torch.float64, device=dev)
    E = torch.zeros(1, dtype=torch.float64, device=dev)
    R_host = torch.empty(NP, NP, dtype=torch.float64).pin_memory()
    yard = yardstick(thc, torch, dev) if rank == 0 else {}
    stream_info = None
    if bvv_mode == "host" and not sharded:
        # B_vv streamed from pinned host memory (3-index arrays live in host memory and are transferred
        # piecewise): time the SAME evaluation with B_vv resident first, in this process, so that the penalty of the
        # stream and the share of it that hides under the GEMMs can be stated.
        bvv_dev = host[5].to(dev)
        hr = thc.thc_setup(o, v, NL, NP, NX, bvv_mode="device")
        dr = list(d)
        dr[5] = bvv_dev
        for _ in range(2):
            hr.thc_residual(*dr, out=R)
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record()
        for _ in range(2):
            hr.thc_residual(*dr, out=R)
            hr.thc_energy_device(dr[0], dr[1], dr[2], dr[3], out=E)
        eb.record(); eb.synchronize()
        resident_ms = ea.elapsed_time(eb) / 2
        bL_r = hr.blocks["bL"]
        hr.close()
        del dr
        # standalone H2D rate of one L-block copy (what one cudaMemcpyAsync of the stream achieves on this link)
        blk = bvv_dev[:bL_r]
        best = 1e30
        for _ in range(4):
            ea.record(); blk.copy_(host[5][:bL_r], non_blocking=True); eb.record(); eb.synchronize()
            best = min(best, ea.elapsed_time(eb))
        h2d_gbs = blk.numel() * 8 / (best * 1e-3) / 1e9
        del blk, bvv_dev
        torch.cuda.empty_cache()
        stream_info = {"bytes_streamed_per_eval": NL * v * v * 8, "h2d_gbs_one_block_standalone": h2d_gbs,
                       "resident_ms_per_step": resident_ms}
    h = thc.thc_setup(o, v, NL, NP, NX, bvv_mode=bvv_mode)
    flops = h.algorithmic_flops
    alg_work = h.algorithmic_work
    input_bytes = sum(t.numel() * 8 for t in host if torch.is_tensor(t))
    use_flush = input_bytes < (512 << 20)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if use_flush else None     # > 126 MB L2
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

    # ---- warm-up (the last warm-up step is profiled per kernel class and finds the dominant class) ----
    # (config 4 takes ~13 minutes per evaluation: its profiles/ lines are taken with --warmup 1 --steps 1)
    W = args.warmup if args.config >= 4 else max(3, args.warmup)
    W = max(1, W)
    for _ in range(W - 1):
        step()
    h.thc_profile_begin(7)
    step()
    prof_w = h.thc_profile_end()
    work_w = h.thc_profile_work()        # EXECUTED flop (gemm, triple) / algorithmic HBM bytes (ew) of that step
    if args.trace and rank == 0:
        with open(args.trace, "w") as f:
            f.write("class,ms,work,rate_T_per_s,description\n")
            for cls, ms, work, desc in h.thc_profile_launches():
                f.write(f"{cls},{ms:.4f},{work:.6g},{work / max(ms, 1e-9) / 1e9:.3f},\"{desc}\"\n")
    dominant = max(prof_w, key=lambda k: prof_w[k][0])
    dom_bit = {"gemm": 1, "triple": 2, "ew": 4}[dominant]

    # ---- timed region: K steps, device-timed per step, L2 flushed between steps when the inputs fit L2 ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    K = args.steps
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    launches0 = h.kernel_launches
    barrier()
    wall0 = time.perf_counter()
    # launch-bound shapes replay a CUDA graph (thc_options.use_graph auto): per-launch events would switch the graph off, so
    # their class times come from the profiled warm-up step instead of the timed region
    live_profile = flops >= 2e10 or sharded
    if live_profile:
        h.thc_profile_begin(dom_bit)
    for k in range(K):
        if use_flush:
            flush.fill_(k & 0xFF)
        ev[k][0].record()
        step()
        ev[k][1].record()
    if live_profile:
        prof = h.thc_profile_end()       # synchronises the stream
    else:
        prof = {k2: (prof_w[k2][0] * K, prof_w[k2][1] * K) for k2 in prof_w}
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
    blocks = h.blocks

    # ---- end to end through thc_residual_host: pinned host buffers in, R + E back on the host, every step ----
    # The device-resident copies of the inputs are released first: the host entry stages its own copies inside the
    # workspace, so its handle is set up with a cap that leaves room for them (same memory budget as above).
    # Same L2 treatment as the device-timed leg (flush before each step when the inputs fit L2, outside the timer).
    # (N > 1: the sharded evaluation has no host-buffer entry; its inputs are copied H2D explicitly every step.)
    e2e_value, Ke = None, 0
    if not args.no_e2e:
        if not sharded:
            h.close()
            del d
            torch.cuda.empty_cache()
            free_b, _ = torch.cuda.mem_get_info(dev)
            cap = int(0.92 * free_b) - input_bytes - NP * NP * 8 - (64 << 20)
            he = thc.thc_setup(o, v, NL, NP, NX, bvv_mode=bvv_mode, workspace_bytes_max=max(cap, 1 << 28))

        def e2e_step():
            if sharded:
                dh = [t.to(dev, non_blocking=True) if torch.is_tensor(t) else t for t in host]
                be = CudaBackend(h, *dh)
                R_host.copy_(residual_sharded(be), non_blocking=True)
                Eh = energy_sharded(be).cpu()
                torch.cuda.synchronize()
                return float(Eh[0])
            return he.thc_residual_host(*host, R_host)       # synchronous

        Ke = max(1, min(K, 5 if args.config == 2 else (1 if args.config >= 3 else K)))
        if args.config <= 2:
            e2e_step()                                        # warm-up of the host entry (workspace allocation)
        barrier()
        e2e_t = 0.0
        for k in range(Ke):
            if use_flush:
                flush.fill_(k & 0xFF)
                torch.cuda.synchronize()
            t0 = time.perf_counter()
            e2e_step()
            e2e_t += time.perf_counter() - t0
        barrier()
        e2e_s = torch.tensor([e2e_t], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
        e2e_value = (1 if sharded else world) * Ke / float(e2e_s.item())
        if not sharded:
            he.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines: ALGORITHMIC work / measured class time; executed work as a separate ratio ----
    pk = measured_peaks()
    tensor_peak = pk["bf16"] * NOMINAL_FP64_TENSOR_OVER_BF16
    alu_peak = SMS * DFMA_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    spec = {"gemm": ("tensor", "TFLOP/s", tensor_peak, 1e12,
                     f"{pk['source']} bf16 burst {pk['bf16']:.1f} TFLOP/s x nominal FP64-tensor/bf16 ratio 45/2250"),
            "triple": ("alu", "TFLOP/s", alu_peak, 1e12,
                       f"148 SMs x 64 FP64 FMA lanes x 2 flop x {pk['sm_max_mhz']:.0f} MHz (max SM clock, {pk['source']})"),
            "ew": ("hbm", "GB/s", pk["hbm"], 1e9, f"{pk['source']} copy bandwidth")}
    names = {"gemm": "dgemm kernels (FP64 DMMA, all GEMM chains)", "triple": "triple_product_kernel (Alg.6 line 11)",
             "ew": "Hadamard / reduction kernels"}

    def class_roof(cls, ms, launches_n, executed):
        bound, unit, peak, scale, src = spec[cls]
        # ew: the class's work is HBM bytes (every operand element once per launch), identical executed / algorithmic
        alg = executed if cls == "ew" else alg_work[cls]
        ach = alg / (ms * 1e-3) / scale if ms > 0 else None
        r = {"bound": bound, "kernel": names[cls], "achieved": ach, "peak": peak, "unit": unit, "peak_source": src,
             "frac": ach / peak if ach else None, "ms": ms, "launches": launches_n,
             "algorithmic_work": alg, "executed_over_algorithmic": executed / alg if alg else None}
        return r

    dom_ms, dom_n = prof[dominant]
    roof = class_roof(dominant, dom_ms / K, dom_n / K, work_w[dominant])
    roof["traffic"] = ncu_traffic(args.config, dominant)
    roof["launches_per_step"] = roof.pop("launches")
    roof["ms_per_step"] = roof.pop("ms")
    roof["share_of_step"] = roof["ms_per_step"] / (1e3 * total_s / K)
    roof["class_ms_warmup_step"] = {k: round(prof_w[k][0], 4) for k in prof_w}
    roof["timed_in"] = "timed region (CUDA events around every launch of the class)" if live_profile else \
        "profiled warm-up step (the timed region replays a CUDA graph)"
    per_class = {k: class_roof(k, prof_w[k][0], prof_w[k][1], work_w[k]) for k in prof_w if prof_w[k][0] > 0}
    for k in per_class:
        per_class[k].pop("kernel"); per_class[k].pop("peak_source")
        per_class[k]["share_of_step"] = per_class[k]["ms"] / sum(prof_w[j][0] for j in prof_w)
    if "gemm" in per_class:
        per_class["gemm"]["frac_of_sustained_peak"] = per_class["gemm"]["achieved"] / (pk["bf16_sustained"] * NOMINAL_FP64_TENSOR_OVER_BF16)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": 1e3 * total_s / K, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config{args.config}", "o": o, "v": v, "NL": NL, "NP": NP, "NX": NX, "seed": c["seed"],
                       "blocks": blocks, "l2": "flushed between steps (256 MiB write), both legs" if use_flush else "inputs larger than L2",
                       "parallelism": "1 GPU" if world == 1 else f"one evaluation sharded over {world} GPUs (Cholesky ranges + T2^2 row blocks, one all-reduce)",
                       "B_vv": {"provider": "provider callback, generated per L-block on the device",
                                "host": "pinned host memory, streamed per L-block", "device": "resident in HBM"}[bvv_mode]},
            "tflops_fp64_algorithmic": (1 if sharded else world) * flops * K / total_s / 1e12,
            "algorithmic_flops_per_eval": flops, "energy_Eh": E_val,
            "wall_s_timed_region": wall, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": input_bytes, "d2h_bytes_per_step": NP * NP * 8 + 8,
                    "steps": Ke},
            "gpu_launches": launches, "roofline": roof, "rooflines_by_class": per_class,
            "extra": {"yardstick": yard}}
    if stream_info:
        t_copy_ms = stream_info["bytes_streamed_per_eval"] / (stream_info["h2d_gbs_one_block_standalone"] * 1e9) * 1e3
        penalty_ms = 1e3 * total_s / K - stream_info["resident_ms_per_step"]
        stream_info.update({"streamed_ms_per_step": 1e3 * total_s / K, "penalty_ms_per_step": penalty_ms,
                            "copy_ms_if_not_overlapped": t_copy_ms,
                            "fraction_of_copy_hidden": max(0.0, min(1.0, 1.0 - penalty_ms / t_copy_ms)),
                            "effective_h2d_gbs_over_step": stream_info["bytes_streamed_per_eval"] / total_s * K / 1e9})
        line["extra"]["bvv_stream"] = stream_info
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(args.config)
    print(json.dumps(line), flush=True)
    if sharded:
        h.close()
    if world > 1:
        dist.destroy_process_group()


def run_second_workload(args):
    """--workload second: the two appendix set-up steps at the dimensions of config C, timed with CUDA
    events after 3 warm-ups, with the per-class split of the library's own launch timers.  mp2_density: thc_mp2_density on
    (Xo, Xv, Z) of the config.  als_update: thc_cp_als_update on a projector-shaped array (U^P_ia), A[I = NP][J = o][K = v]
    with N = NP factors and 10 PCG iterations.  Flop counts are those of the evaluation order in DESIGN.md section 6.8
    (FMA = 2 flop, no padding).  One JSON line; not the BASELINE metric."""
    import torch
    import paper_2111_11473_b200 as thc
    from thc_synth import CONFIGS
    from thc_synth import device as synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --workload second: no CUDA device")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    c = CONFIGS[args.config]
    o, v, NL, NP, NX = c["o"], c["v"], c["NL"], c["NP"], c["NX"]
    K, W = max(1, args.steps), max(3, args.warmup)
    pk = measured_peaks()
    tensor_peak = pk["bf16"] * NOMINAL_FP64_TENSOR_OVER_BF16
    h = thc.thc_setup(o, v, 4, NP, 16)
    g = torch.Generator(device=dev).manual_seed(c["seed"])

    def rnd(*shape, scale=1.0):
        return torch.randn(*shape, dtype=torch.float64, device=dev, generator=g) * scale

    def timed(fn):
        for _ in range(W):
            fn()
        h.thc_profile_begin(7)
        fn()
        prof, work = h.thc_profile_end(), h.thc_profile_work()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = h.kernel_launches
        a.record()
        for _ in range(K):
            fn()
        b.record()
        b.synchronize()
        return a.elapsed_time(b) / K, prof, work, (h.kernel_launches - l0) // K

    def report(ms, prof, work, launches, flops):
        cls = {}
        if prof["gemm"][0] > 0:
            ach = work["gemm"] / (prof["gemm"][0] * 1e-3) / 1e12
            cls["gemm"] = {"bound": "tensor", "ms": prof["gemm"][0], "launches": prof["gemm"][1], "achieved": ach,
                           "peak": tensor_peak, "unit": "TFLOP/s", "frac": ach / tensor_peak}
        if prof["ew"][0] > 0:
            ach = work["ew"] / (prof["ew"][0] * 1e-3) / 1e9
            cls["ew"] = {"bound": "hbm", "ms": prof["ew"][0], "launches": prof["ew"][1], "achieved": ach, "peak": pk["hbm"],
                         "unit": "GB/s", "frac": ach / pk["hbm"]}
        return {"ms": ms, "flops": flops, "tflops_fp64": flops / (ms * 1e-3) / 1e12, "gpu_launches": launches,
                "executed_gemm_flops_over_counted": work["gemm"] / flops, "rooflines_by_class": cls}

    Xo, Xv = rnd(o, NP, scale=NP ** -0.5), rnd(v, NP, scale=NP ** -0.5)
    Z = rnd(NP, NP, scale=0.1)
    Z = 0.5 * (Z + Z.T)
    f_mp2 = (2.0 * NP * NP * (o + v) + 4.0 * NP ** 3 + 2.0 * (o + v) * NP * NP + 2.0 * (o * o + v * v) * NP
             + 6.0 * o * v * NP * NP + 4.0 * o * NP ** 3 + 2.0 * o * NP * NP + 2.0 * o * o * NP + 2.0 * o * v * v * NP)
    out = {"workload": "second (SURVEY.md 8(f)-4)", "config": {"workload": f"config{args.config} dimensions", "o": o, "v": v, "NP": NP},
           "steps": K, "warmup": W, "dtype": "f64", "data": "synthetic"}
    out["mp2_density"] = report(*timed(lambda: h.thc_mp2_density(Xo, Xv, Z)), f_mp2)
    del Z
    I, J, Kk, N, iters = NP, o, v, NP, 10
    A = rnd(I, J, Kk)
    Yf, Zf, Xf = rnd(J, N), rnd(Kk, N), rnd(I, N)
    f_als = 2.0 * N * N * (J + Kk) + 2.0 * I * J * Kk * N + 2.0 * I * N * N * (iters + 1)
    out["als_update"] = report(*timed(lambda: h.thc_cp_als_update(A, Yf, Zf, Xf, iters)), f_als)
    out["als_update"]["shape"] = {"I": I, "J": J, "K": Kk, "N": N, "pcg_iters": iters}
    h.close()
    print(json.dumps(out), flush=True)


def run_probe(args):
    """Measured ceilings of this device for the FP64 kernels (thc_probe in the library): DMMA and DFMA issue rates,
    both interleaved, shared-memory -> register bandwidth by access width."""
    import torch
    import paper_2111_11473_b200 as thc
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --probe: no CUDA device")
    h = thc.thc_setup(4, 8, 4, 16, 16)
    out = {"probe": h.thc_probe(), "device": torch.cuda.get_device_name(0)}
    out["yardstick"] = yardstick(thc, torch, torch.device("cuda", 0))
    h.close()
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--bvv", default=None, choices=["device", "host", "provider"],
                    help="where B_vv lives (default: device; provider at config 4)")
    ap.add_argument("--trace", default=None, help="write the per-launch records of the profiled warm-up step to this CSV")
    ap.add_argument("--probe", action="store_true")
    ap.add_argument("--workload", default="residual", choices=["residual", "second"],
                    help="second = the appendix set-up steps (thc_mp2_density, thc_cp_als_update) at the config's dimensions")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end (host buffers) leg")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.probe:
        run_probe(args)
    elif args.workload == "second":
        run_second_workload(args)
    else:
        if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
            respawn_under_torchrun(args)
        run_ours(args)


if __name__ == "__main__":
    main()
