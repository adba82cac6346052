#!/usr/bin/env python
"""pacc_sweep.py -- Metropolis acceptance P_acc of the bMPS proposal over L, chi, beta (the quantity of the
paper's Fig. 3), on seeded synthetic +-J instances.

    python pacc_sweep.py [--Ls 8,16,...] [--chis 8,16] [--betas 0.66,1.0,1.5] [--n-dis 32] [--n-samples 256]
                         [--prec f64|f32|f32s] [--out gpurun_out/pacc.jsonl]

One JSON line per (L, chi, beta): P_acc = accepted / (n_dis (n_s - 1)) (reading G15 of DESIGN.md), the mean of
min(1, ratio), seconds per phase.  Everything runs through the C ABI binding; nothing here touches oracle/."""
import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from tnmc_workloads import make_couplings  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--Ls", default="8,16,32,64,128,256,512,1024")
    ap.add_argument("--chis", default="8,16")
    ap.add_argument("--betas", default="0.66,1.0,1.5")
    ap.add_argument("--n-dis", type=int, default=32)
    ap.add_argument("--n-samples", type=int, default=256)
    ap.add_argument("--prec", default="f64", choices=["f64", "f32", "f32s", "tf32"])
    ap.add_argument("--inst-seed", type=int, default=3003)
    ap.add_argument("--seed", type=int, default=4004)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    import torch
    from paper_2509_19006_b200 import tnmc
    if not torch.cuda.is_available():
        raise SystemExit("pacc_sweep.py needs a CUDA device (no CPU fallback)")
    dev = torch.device("cuda:0")
    prec = {"f64": tnmc.TNMC_F64, "f32": tnmc.TNMC_F32_LOGSCALE, "f32s": tnmc.TNMC_F32_STORE, "tf32": tnmc.TNMC_TF32_FAST}[a.prec]
    out = open(a.out, "a") if a.out else None
    for L in [int(x) for x in a.Ls.split(",")]:
        n_dis = a.n_dis
        n_s = a.n_samples if L < 1024 else min(a.n_samples, 128)
        Jr, Jd = make_couplings(L, n_dis, a.inst_seed)
        Jr_d, Jd_d = torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev)
        for chi in [int(x) for x in a.chis.split(",")]:
            # full stack while it fits comfortably, else two-level checkpoints with stride ~ sqrt(L)
            P = 8 if chi <= 8 else (16 if chi <= 16 else 32)
            full_bytes = n_dis * L * L * 2 * P * P * (8 if a.prec == "f64" else 4)
            ckpt = 0 if full_bytes < 60e9 else max(2, int(round(L ** 0.5)))
            for beta in [float(x) for x in a.betas.split(",")]:
                ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
                ctx = tnmc.Context(L, chi, beta, Jr_d, Jd_d, n_s, prec=prec, ckpt_stride=ckpt)
                ev[0].record(); logZ = ctx.tnmc_build_envs()
                ev[1].record(); bits, logq = ctx.tnmc_sample(n_s, a.seed)
                ev[2].record(); E = ctx.tnmc_energy(bits)
                acc, n_acc, _, smin = ctx.tnmc_metropolis(E, logq, a.seed, want_sum_min1=True)
                ev[3].record()
                torch.cuda.synchronize()
                flags = ctx.tnmc_get_flags()
                rec = {"L": L, "chi": chi, "beta": beta, "n_dis": n_dis, "n_samples": n_s, "prec": a.prec, "ckpt_stride": ckpt,
                       "p_acc": float(n_acc.sum()) / (n_dis * (n_s - 1)),
                       "mean_min1_ratio": float(smin.sum()) / (n_dis * (n_s - 1)),
                       "p_acc_min_over_disorders": float(n_acc.min()) / (n_s - 1),
                       "logZ_per_site_mean": float(logZ.mean()) / (L * L),
                       "build_s": ev[0].elapsed_time(ev[1]) * 1e-3, "sample_s": ev[1].elapsed_time(ev[2]) * 1e-3,
                       "flags": {k: v for k, v in flags.items() if v and k not in ("sigma_zero", "near_threshold")},
                       "when": time.strftime("%Y-%m-%dT%H:%M:%S")}
                line = json.dumps(rec)
                print(line, flush=True)
                if out:
                    out.write(line + "\n")
                    out.flush()
                ctx.close()
                del ctx, bits, logq, E, acc
                torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
