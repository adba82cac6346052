#!/usr/bin/env python
"""bench.py -- accepted samples/s of the BatchTNMC hot path on synthetic +-J instances.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3|C2|C4s|C5s|...] [--impl ours|reference]

Default workload: C3 (BASELINE.json configs[2], 128x128, chi=32, 256 disorders x 256 samples, FP64) -- the largest
config whose whole step fits the default run (chi = 32 is the bond dimension of three of the five configs, the
paper's 1024^2 run included); C2 and the slices of C4/C5 are behind --workload.

A "step" is one pass of the whole hot path over one batch: tnmc_create (pack couplings) ->
tnmc_build_envs -> tnmc_sample -> tnmc_energy -> tnmc_metropolis for every beta of the workload.
`value` times the device-resident path (couplings already in HBM); `e2e` times tnmc_run_host with
pinned HOST buffers (H2D of the couplings and D2H of configurations, E, log q, flags inside the
timed region).  One JSON line on stdout (rank 0).  See DESIGN.md, "Measurement".
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
sys.path.insert(0, ROOT)

from tnmc_workloads import CONFIGS, make_couplings, make_gaussian_couplings  # noqa: E402

# name -> (config key, n_dis, n_samples, ckpt_stride, note).  C3 (BASELINE.json configs[2]) is the
# default; C2 is configs[1]; C4s / C5s are disorder x sample SLICES of configs[3] / configs[4] sized to
# finish in minutes (the full configs are chunked runs of the same calls).
WORKLOADS = {
    "C1": ("C1", None, None, 0, "configs[0] 8x8 chi=16 exact"),
    "C2": ("C2", None, None, 0, "configs[1] 32x32 chi=16 100x100 beta in {0.5,1,2}"),
    "C3": ("C3", None, None, 0, "configs[2] 128x128 chi=32 256x256 FP64"),
    "C3q": ("C3q", None, None, 0, "profiling shape of configs[2]: 64x64 chi=32 256x256 (C3's kernels and grid at a quarter of the rows and columns)"),
    "C4s": ("C4", 148, 200, 23, "configs[3] 512x512 chi=32, slice of 148 disorders x 200 samples, checkpoint stride 23"),
    "C5s": ("C5", 74, 128, 32, "configs[4] 1024x1024 chi=32, slice of 74 disorders x 128 samples, checkpoint stride 32"),
    # the full configs[3] / configs[4]: disorder chunks of the same calls, one after the other in the same workspace
    "C4": ("C4", None, None, 23, "configs[3] 512x512 chi=32, 500 disorders x 200 samples in 2 chunks of 250 disorders, checkpoint stride 23", 250),
    "C5": ("C5", None, None, 32, "configs[4] 1024x1024 chi=32, 1000 disorders x 1000 samples in 10 chunks of 100 disorders (152 GB of HBM per chunk), checkpoint stride 32", 100),
    "C5c": ("C5", 100, 1000, 32, "configs[4] 1024x1024 chi=32: ONE of the ten 100-disorder chunks of C5 (100 disorders x 1000 samples, 152 GB of HBM), checkpoint stride 32"),
    "C5pf": ("C5p", None, None, 32, "the paper headline setting IN FULL (PAPER.md:286: 1024x1024, chi=8, 1000 disorders x 1000 samples) in 4 chunks of 250 disorders, checkpoint stride 32; run it with --prec f32 for the paper's precision class", 250),
    "C5c148": ("C5", 148, 1000, 32, "configs[4] 1024x1024 chi=32: a chunk of 148 disorders x 1000 samples (one CTA per SM in the build); fits HBM only with --prec f32s (FP32 stack, FP64 arithmetic), checkpoint stride 32"),
    "C5p": ("C5p", 500, 400, 32, "the paper headline setting (1024x1024, chi=8, PAPER.md:286) in FP64: slice of 500 disorders x 400 samples (one fifth of its 10^6 proposals), checkpoint stride 32"),
}
SLICES = ("C4s", "C5s", "C5c", "C5c148", "C5p", "C5pf", "C4", "C5")   # steps of minutes to hours: --warmup is taken as given (0 allowed; said in config)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--prec", default="f64", choices=["f64", "f32", "f32s", "tf32"],
                    help="f64: the parity path; f32: TNMC_F32_LOGSCALE (FP32 stack, 3xTF32 tensor-core sampler, FP64 compression); tf32: TNMC_TF32_FAST (plain TF32 products); "
                         "f32s: TNMC_F32_STORE (FP32 stack, all arithmetic FP64)")
    ap.add_argument("--chunk", type=int, default=0, help="disorders per chunk (overrides the workload's; 0 = its default)")
    ap.add_argument("--couplings", default="pmj", choices=["pmj", "gaussian"],
                    help="pmj: +-J (the BASELINE configs); gaussian: J ~ N(0,1) through tnmc_create_real (no e2e / cpu_baseline leg)")
    ap.add_argument("--ckpt", type=int, default=-1, help="checkpoint stride (overrides the workload's; -1 = its default, 0 = full stack)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def workload(name):
    key, n_dis, n_s, ckpt, note = WORKLOADS[name][:5]
    c = dict(CONFIGS[key])
    c["chunk"] = WORKLOADS[name][5] if len(WORKLOADS[name]) > 5 else None
    if n_dis:
        c["n_dis"] = n_dis
    if n_s:
        c["n_samples"] = n_s
    c["ckpt"] = ckpt
    c["note"] = note
    return c


# ------------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi, during the timed region)
# ------------------------------------------------------------------------------------------------
class Clocks:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.stop = index, [], threading.Event()
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


# ------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores
# ------------------------------------------------------------------------------------------------
def oracle_disorder(c, beta, d, n_so):
    """The oracle's whole path for ONE disorder and n_so proposals: (seconds of the build, seconds of everything
    per-proposal -- uniforms, sampling, energies, Metropolis scan --, accepted count)."""
    from oracle import bmps, exact, metropolis, philox, sampler
    L, chi = c["L"], c["chi"]
    Jr, Jd = make_couplings(L, 1, c["inst_seed"], first_disorder=d)
    Jr, Jd = Jr[0], Jd[0]
    t0 = time.perf_counter()
    cache, ls = bmps.build_cache(Jr, Jd, beta, chi)
    bmps.log_z(cache[0], ls[0])
    t1 = time.perf_counter()
    samples = np.arange(n_so)
    u = philox.spin_uniforms(c["seed"], d, samples[:, None], np.arange(L * L)[None, :]).reshape(n_so, L, L)
    cfg, logq, _ = sampler.sample(cache, Jd, beta, u)
    E = exact.energy(cfg, Jr, Jd)
    um = philox.metropolis_uniforms(c["seed"], d, samples)
    _, n_acc, *_ = metropolis.metropolis_scan(E, logq, beta, um)
    return t1 - t0, time.perf_counter() - t1, int(n_acc)


def oracle_n_so(c):
    """proposals per disorder of the bounded oracle sample: the workload's own count where the oracle's sampler
    finishes them in seconds (L <= 64), 16 beyond (its cost is then projected, see oracle_step)"""
    return c["n_samples"] if c["L"] <= 64 else min(c["n_samples"], 16)


def oracle_step(c, budget_s, first_d=0):
    """One bounded sample of the workload on the host: disorders first_d, first_d+1, ... through every beta until
    budget_s seconds are used (at least one disorder).  Returns the PROJECTED accepted samples/s of the workload
    -- the build is paid once per disorder whatever the number of proposals, so the rate at the workload's own
    n_samples is  p_acc * n_samples / (t_build + n_samples * t_per_proposal)  per (disorder, beta), with t_build,
    t_per_proposal and p_acc measured on the sample --, the seconds spent, the disorders used and a description."""
    n_so, n_s = oracle_n_so(c), c["n_samples"]
    tb = tp = 0.0
    acc = nd = 0
    t0 = time.perf_counter()
    while nd < c["n_dis"] and (nd == 0 or time.perf_counter() - t0 < budget_s):
        for beta in c["betas"]:
            b, p, a = oracle_disorder(c, beta, first_d + nd, n_so)
            tb += b
            tp += p
            acc += a
        nd += 1
    units = nd * len(c["betas"])
    p_acc = acc / (units * max(n_so - 1, 1))
    t_build, t_prop = tb / units, tp / (units * n_so)
    value = p_acc * (n_s - 1) / (t_build + n_s * t_prop)
    desc = (f"{nd} disorder(s) x {n_so} proposals x {len(c['betas'])} beta(s), whole path (build, uniforms, sampling, energy, "
            f"Metropolis); measured per (disorder, beta): build {t_build:.2f} s, {1e3 * t_prop:.1f} ms per proposal, p_acc {p_acc:.4f}; "
            f"value = p_acc (n_s - 1) / (t_build + n_s t_proposal) at the workload's n_s = {n_s}")
    return value, time.perf_counter() - t0, nd, desc


def cpu_info():
    """what the oracle actually runs on: one Python thread issuing numpy/LAPACK calls on matrices of at most
    4 chi x 4 chi; the BLAS pool is reported beside it because it exists, not because it is used at that size"""
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    pool = 1
    try:
        from threadpoolctl import threadpool_info
        pool = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        pass
    return {"cores": 1, "cpu_model": model, "host_cores": os.cpu_count() or 1, "blas_pool_threads": pool,
            "parallelism": "1 process, 1 Python thread; LAPACK/BLAS calls on <= 128x128 matrices run effectively on one core"}


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c = workload(args.workload)
    # the whole run is meant to end within a few minutes: ~200 s of oracle time over the K timed steps, never
    # less than one disorder per step; one warm-up step at most (host code: nothing to warm beyond imports)
    budget = max(2.0, 200.0 / max(args.steps, 1))
    n_warm = min(args.warmup, 1)
    for _ in range(n_warm):
        oracle_step(c, 0.0)
    vals, tot_t, nd_tot, desc = [], 0.0, 0, ""
    for _ in range(args.steps):
        v, dt, nd, desc = oracle_step(c, budget, first_d=nd_tot % c["n_dis"])
        vals.append(v)
        tot_t += dt
        nd_tot += nd
    val = float(np.mean(vals))
    info = cpu_info()
    line = {"impl": "reference", "metric": "accepted samples/s", "value": val, "unit": "samples/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": n_warm, "warmup_requested": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": bench_config(args.workload, c),
            "cpu_baseline": dict(value=val, unit="samples/s", kind="oracle", sample="per step: " + desc, **info),
            "e2e": {"value": val, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def bench_config(name, c):
    """the keys both arms print for the same workload"""
    return {"workload": name, "note": c["note"], "L": c["L"], "chi": c["chi"], "betas": list(c["betas"]),
            "n_dis_per_gpu": c["n_dis"], "n_samples": c["n_samples"], "ckpt_stride": c["ckpt"],
            "l2": "GPU arm: flushed (256 MiB memset) before every timed step, in the value loop and in the e2e loop, and the env "
                  "stack is larger than L2; reference arm: host only"}


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def main_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_19006_b200 import model, shard, tnmc

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    c = workload(args.workload)
    if args.ckpt >= 0:
        c["ckpt"] = args.ckpt
    L, chi, n_dis, n_s, ckpt = c["L"], c["chi"], c["n_dis"], c["n_samples"], c["ckpt"]
    n_dis_total = n_dis                                   # per rank
    if args.chunk:
        c["chunk"] = args.chunk
    if c.get("chunk"):
        n_dis = min(c["chunk"], n_dis_total)              # buffers and contexts are sized for one chunk
    chunks = [(c0, min(n_dis, n_dis_total - c0)) for c0 in range(0, n_dis_total, n_dis)]
    P = model.pad_chi(chi)
    betas = list(c["betas"])
    # weak scaling: every rank owns its own n_dis disorders (global indices rank*n_dis ...); no collective on the data path
    first = shard.first_disorder(rank, n_dis_total)
    real_j = args.couplings == "gaussian"
    if real_j:
        args.no_e2e = args.no_cpu_baseline = True          # tnmc_run_host and the timed oracle leg are +-J only
    gen = make_gaussian_couplings if real_j else make_couplings
    Jr_np, Jd_np = gen(L, n_dis_total, c["inst_seed"], first_disorder=first)
    Jr_h, Jd_h = torch.from_numpy(Jr_np).pin_memory(), torch.from_numpy(Jd_np).pin_memory()
    Jr, Jd = Jr_h.to(dev), Jd_h.to(dev)
    prec = {"f64": tnmc.TNMC_F64, "f32": tnmc.TNMC_F32_LOGSCALE, "f32s": tnmc.TNMC_F32_STORE, "tf32": tnmc.TNMC_TF32_FAST}[args.prec]
    need = tnmc.tnmc_workspace_bytes(L, chi, n_dis, n_s, prec=prec, ckpt_stride=ckpt)
    if real_j:
        need = int(tnmc.lib.tnmc_workspace_bytes_real(L, chi, n_dis, n_s, prec, ckpt))
    need_h = tnmc.tnmc_run_host_workspace_bytes(L, chi, n_dis, n_s, prec=prec, ckpt_stride=ckpt)
    W = tnmc.words(L)
    nb = len(betas)
    # the betas of a step are independent problems: each gets its own stream, workspace and outputs, and
    # the nb launches of every phase run side by side (fork/join on events around each phase)
    stream = torch.cuda.current_stream()
    streams = [stream] + [torch.cuda.Stream(device=dev) for _ in range(nb - 1)]
    ws = [torch.empty(max(need, need_h), dtype=torch.uint8, device=dev) for _ in betas]
    bits = [torch.empty((n_dis, n_s, L, W), dtype=torch.int32, device=dev) for _ in betas]
    logq = [torch.empty((n_dis, n_s), dtype=torch.float64, device=dev) for _ in betas]
    E = [torch.empty((n_dis, n_s), dtype=torch.float64 if real_j else torch.int32, device=dev) for _ in betas]
    logZ = [torch.empty(n_dis, dtype=torch.float64, device=dev) for _ in betas]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    ev = lambda: torch.cuda.Event(enable_timing=True)
    PHASES = ("build", "sample", "energy", "metropolis")
    flag_tot = {}

    def step(timed):
        """one pass over the batch (all disorder chunks, one after the other); returns (accepted, launches, phase ms dict)"""
        acc, launches = 0, 0
        ph = {k: 0.0 for k in PHASES}
        for c0, nd in chunks:
            a1, l1, p1 = step_chunk(c0, nd)
            acc += a1
            launches += l1
            for k in PHASES:
                ph[k] += p1[k]
        return acc, launches, ph

    def step_chunk(c0, nd):
        ctxs, n_accs = [None] * nb, [None] * nb
        Jr_c, Jd_c = Jr[c0:c0 + nd], Jd[c0:c0 + nd]

        def run(phase, i):
            if phase == "build":
                ctxs[i] = tnmc.Context(L, chi, betas[i], Jr_c, Jd_c, n_s, first_disorder=first + c0, prec=prec, ckpt_stride=ckpt, workspace=ws[i])
                ctxs[i].tnmc_build_envs(logZ[i][:nd])
            elif phase == "sample":
                ctxs[i].tnmc_sample(n_s, c["seed"], cfg_bits=bits[i][:nd], logq=logq[i][:nd])
            elif phase == "energy":
                ctxs[i].tnmc_energy(bits[i][:nd], E=E[i][:nd])
            else:
                _, n_accs[i], _, _ = ctxs[i].tnmc_metropolis(E[i][:nd], logq[i][:nd], c["seed"])

        e = [ev() for _ in range(len(PHASES) + 1)]
        e[0].record(stream)
        for k, phase in enumerate(PHASES):
            for i, s in enumerate(streams):
                if i > 0:
                    s.wait_event(e[k])
                with torch.cuda.stream(s):
                    run(phase, i)
            for s in streams[1:]:
                done = torch.cuda.Event()
                done.record(s)
                stream.wait_event(done)
            e[k + 1].record(stream)
        torch.cuda.synchronize()
        acc = sum(int(n.sum().item()) for n in n_accs)
        launches = sum(cx.tnmc_launch_count() for cx in ctxs)
        ph = {k: e[i].elapsed_time(e[i + 1]) for i, k in enumerate(PHASES)}
        for cx in ctxs:
            for k, v in cx.tnmc_get_flags().items():       # device fault / near-threshold counters of this pass
                flag_tot[k] = flag_tot.get(k, 0) + v
            cx.close()
        return acc, launches, ph

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    n_warm = args.warmup if args.workload in SLICES else max(args.warmup, 3)
    for _ in range(n_warm):
        step(False)
    phases = {"build": 0.0, "sample": 0.0, "energy": 0.0, "metropolis": 0.0}
    tot_ms, tot_acc, tot_launch = 0.0, 0, 0
    flag_tot.clear()                                        # counters of the timed steps only
    with Clocks(local_rank) as clk:
        for _ in range(args.steps):
            flush.zero_()                                   # L2 flush between timed iterations
            barrier()
            e0, e1 = ev(), ev()
            e0.record(stream)
            acc, launches, ph = step(True)
            e1.record(stream)
            barrier()
            tot_ms += e0.elapsed_time(e1)
            tot_acc += acc
            tot_launch += launches
            for k in phases:
                phases[k] += ph[k]
    ms_total, acc_total = shard.reduce_job(tot_ms, tot_acc, dev)
    value = acc_total / (ms_total * 1e-3)

    # ---- end to end: host buffers through tnmc_run_host, one host thread + stream per beta
    e2e = None
    if not args.no_e2e:
        from concurrent.futures import ThreadPoolExecutor
        outs = [None] * nb

        def host_pass(i):
            torch.cuda.set_device(local_rank)
            tot = 0
            with torch.cuda.stream(streams[i]):
                for c0, nd in chunks:
                    outs[i] = tnmc.tnmc_run_host(L, chi, betas[i], Jr_h[c0:c0 + nd], Jd_h[c0:c0 + nd], n_s, c["seed"], ws[i],
                                                 first_disorder=first + c0, prec=prec, ckpt_stride=ckpt,
                                                 out=outs[i] if len(chunks) == 1 or nd == n_dis else None)
                    tot += int(outs[i]["n_accepted"].sum().item())
            return tot

        with ThreadPoolExecutor(max_workers=nb) as pool:
            for _ in range(1 if args.workload in SLICES else 2):
                list(pool.map(host_pass, range(nb)))
            e_acc = 0
            barrier()
            t0 = time.perf_counter()
            for _ in range(args.steps):
                flush.zero_()                               # same L2 flush as the `value` loop (inside the timed region: ~0.1 ms)
                torch.cuda.synchronize()
                e_acc += sum(pool.map(host_pass, range(nb)))
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
        dt_max, e_acc_sum = shard.reduce_job(dt, e_acc, dev)
        h2d = nb * (Jr_h.numel() + Jd_h.numel())
        d2h = len(chunks) * sum(v.numel() * v.element_size() for o in outs for v in o.values() if v is not None)
        e2e = {"value": e_acc_sum / dt_max, "unit": "samples/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "how": "tnmc_run_host per beta (pinned host buffers; H2D of the couplings, D2H of configurations, E, log q, accepted flags, log Z, counts), "
                      "wall clock over the timed steps, L2 flushed before every step like the `value` loop"}

    if rank == 0:
        # the nb launches of a phase run concurrently: duration of the group, algorithmic work of the group
        build_ms = phases["build"] / args.steps
        sample_ms = phases["sample"] / args.steps
        build_flops = nb * model.build_flops_per_disorder(L, chi) * n_dis_total * (2.0 if ckpt else 1.0)
        peak_dmma = tnmc.tnmc_fp64_peak_tflops(1)
        peak_dfma = tnmc.tnmc_fp64_peak_tflops(0)
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = peaks.get("hbm_gbs", 6650.0)
        hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"

        def matmul_peak(dtype, n, tf32):
            """library GEMM rate on this GPU, TFLOP/s: (burst = best of 10, sustained = back to back for ~1.5 s)"""
            old = torch.backends.cuda.matmul.allow_tf32
            torch.backends.cuda.matmul.allow_tf32 = tf32
            try:
                a = torch.randn(n, n, dtype=dtype, device=dev)
                b = torch.randn(n, n, dtype=dtype, device=dev)
                for _ in range(2):
                    a @ b
                best = 1e30
                for _ in range(10):
                    e0, e1 = ev(), ev()
                    e0.record(); a @ b; e1.record(); e1.synchronize()
                    best = min(best, e0.elapsed_time(e1))
                reps = max(3, int(1500.0 / best))
                e0, e1 = ev(), ev()
                e0.record()
                for _ in range(reps):
                    a @ b
                e1.record(); e1.synchronize()
                sus = e0.elapsed_time(e1) / reps
                return 2.0 * n ** 3 / (best * 1e-3) / 1e12, 2.0 * n ** 3 / (sus * 1e-3) / 1e12
            finally:
                torch.backends.cuda.matmul.allow_tf32 = old

        fp64_mm = matmul_peak(torch.float64, 4096, False)
        tf32_mm = matmul_peak(torch.float32, 8192, True) if args.prec in ("f32", "tf32") else None
        samp_flops = nb * model.sample_flops_per_chain_site(P) * n_dis_total * n_s * L * L
        if args.prec == "f32":
            samp_flops *= 3.0                                   # 3xTF32: three MMAs per product
        w_env = 8 if args.prec == "f64" else 4
        samp_bytes = nb * model.sample_bytes_per_chain_site(P, w=w_env) * n_dis_total * n_s * L * L
        if ckpt:
            # checkpoint mode: tnmc_sample recomputes every segment with build_rows_kernel before sampling it, so the
            # sample phase holds a second full build pass; the build kernel's time is taken as build + sample phase
            # (an upper bound: it includes the sampler's own share) against the flops of both passes
            build_ms += sample_ms
        dominant = "build_rows_kernel" if (ckpt or phases["build"] >= phases["sample"]) else "sample_rows_kernel"

        def ncu_traffic(kernel):
            """DRAM bytes per launch of `kernel` on this workload from the committed ncu --set full capture (profiles/traffic.csv)"""
            try:
                for ln in open(os.path.join(ROOT, "profiles", "traffic.csv")).read().splitlines()[1:]:
                    w_, k_, b_ = ln.split(",")[:3]
                    if w_ == args.workload and k_ == kernel:
                        return int(b_)
            except Exception:
                pass
            return None

        # sampler: which roof it is judged against depends on the arithmetic.  FP64: the DMMA pipe (intensity 4P/8 flop/B
        # is above the FP64 ridge); TF32 modes: HBM (the TF32 tensor roof is ~20x above what the bytes allow)
        samp_tf = samp_flops / (sample_ms * 1e-3) / 1e12
        samp_gbs = samp_bytes / (sample_ms * 1e-3) / 1e9
        if args.prec in ("f64", "f32s"):
            samp_roof = {"bound": "tensor", "kernel": "sample_rows_kernel", "achieved": samp_tf, "peak": peak_dmma, "unit": "TFLOP/s",
                         "frac": samp_tf / peak_dmma, "peak_source": "FP64 DMMA (mma.sync.m8n8k4.f64) rate measured live by tnmc_fp64_peak_tflops(1)",
                         "hbm_gbs": samp_gbs, "frac_hbm_peak": samp_gbs / hbm_peak}
        else:
            samp_roof = {"bound": "hbm", "kernel": "sample_rows_tf32_kernel", "achieved": samp_gbs, "peak": hbm_peak, "unit": "GB/s",
                         "frac": samp_gbs / hbm_peak, "peak_source": hbm_src, "tflops": samp_tf,
                         "tf32_matmul_peak_tflops": {"burst": tf32_mm[0], "sustained": tf32_mm[1], "how": "torch.matmul fp32 8192^3 with TF32 allowed, measured live"},
                         "frac_tf32_peak": samp_tf / tf32_mm[0]}
        samp_roof.update(ms=sample_ms, traffic=ncu_traffic(samp_roof["kernel"]), algorithmic_flops_per_launch_group=samp_flops,
                         algorithmic_bytes_per_launch_group=samp_bytes, launches_per_group=nb,
                         note="checkpoint mode: the phase also holds the segment recomputation (build_rows_kernel)" if ckpt else None)
        ach = build_flops / (build_ms * 1e-3) / 1e12
        build_roof = {"bound": "alu", "kernel": "build_rows_kernel", "achieved": ach, "peak": peak_dfma, "unit": "TFLOP/s", "frac": ach / peak_dfma,
                      "traffic": ncu_traffic("build_rows_kernel"), "ms": build_ms,
                      "peak_source": "FP64 DFMA rate measured live by tnmc_fp64_peak_tflops(0) on this GPU (FP64 has no tcgen05 kind; the DMMA "
                                     "rate, measured the same way, is within 10 % of it)",
                      "algorithmic_flops_per_launch_group": build_flops, "launches_per_group": nb,
                      "flop_count": "nominal: SURVEY 8(d)'s 205 chi^3 per bond-saturated site-row, summed over the actual bond dimensions "
                                    "(model.build_flops_per_disorder); the kernel executes a different mix (block QR, implicit Q, ~5 Jacobi sweeps)"}
        roof = dict(build_roof if dominant == "build_rows_kernel" else samp_roof)
        energy_ms = phases["energy"] / args.steps
        energy_bytes = nb * n_dis_total * n_s * (L * W * 4 + 4)
        roof["other_kernels"] = {
            "sample_rows_kernel": samp_roof, "build_rows_kernel": build_roof,
            "energy_kernel": {"bound": "hbm", "ms": energy_ms, "achieved": energy_bytes / (energy_ms * 1e-3) / 1e9 if energy_ms > 0 else None, "peak": hbm_peak,
                              "unit": "GB/s", "frac": energy_bytes / (energy_ms * 1e-3) / 1e9 / hbm_peak if energy_ms > 0 else None,
                              "algorithmic_bytes_per_launch_group": energy_bytes},
            "peaks": {"fp64_dfma_tflops": peak_dfma, "fp64_dmma_tflops": peak_dmma, "hbm_gbs": hbm_peak, "hbm_source": hbm_src,
                      "fp64_matmul_tflops": {"burst": fp64_mm[0], "sustained": fp64_mm[1], "how": "torch.matmul fp64 4096^3, measured live"},
                      "tf32_matmul_tflops": None if tf32_mm is None else {"burst": tf32_mm[0], "sustained": tf32_mm[1]}},
        }
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            v_o, dt_o, _, desc_o = oracle_step(c, 15.0)
            cpu = dict(value=v_o, unit="samples/s", kind="oracle", seconds=dt_o, sample=desc_o, **cpu_info())
        cfg_line = bench_config(args.workload, dict(c, n_dis=n_dis_total))
        execution = {"couplings": args.couplings, "disorder_chunks": len(chunks), "parallelism": f"dp{world} (disorders sharded, no collective)",
                     "streams": f"{nb} (one per beta; the launches of each phase run concurrently)", "prec": args.prec}
        line = {"metric": "accepted samples/s", "value": value, "unit": "samples/s", "n_gpus": world, "steps": args.steps,
                "warmup": n_warm, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": {"f64": "f64", "f32": "f64 compression + 3xtf32 sampling (fp32 stack)", "f32s": "f64 arithmetic on an fp32 stack", "tf32": "f64 compression + tf32 sampling (fp32 stack)"}[args.prec], "data": "synthetic",
                "config": cfg_line, "execution": execution,
                "chain_sites_per_s": len(betas) * args.steps * n_dis_total * n_s * L * L * world / (ms_total * 1e-3),
                "flags": dict(flag_tot, note="device counters summed over the timed steps of rank 0 (tnmc_get_flags): near_threshold = draws with |u - p| < 1e-9"),
                "proposals_per_s": len(betas) * args.steps * n_dis_total * n_s * world / (ms_total * 1e-3),
                "p_acc": acc_total / (len(betas) * args.steps * n_dis_total * (n_s - 1) * world),
                "phase_ms_per_step": {k: v / args.steps for k, v in phases.items()},
                "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": tot_launch, "clocks": clk.summary()}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse()
    sys.exit(main_reference(a) if a.impl == "reference" else main_ours(a))
