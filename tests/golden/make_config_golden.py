"""Writes tests/golden/config_<NAME>.npz: the ORACLE's outputs for a stated subset of a BASELINE.json config,
at the config's own lattice size (SURVEY.md 8c last paragraph: "a stated subset of disorders x samples for
C3-C5"; all of C2's disorders).  Imports only oracle/, tnmc_workloads and the oracle-only helper
tests/noise_floor.py; nothing here touches the CUDA path.

    python tests/golden/make_config_golden.py C2      # 100 disorders x 3 beta x 32 samples, ~15 min
    python tests/golden/make_config_golden.py C3      # 2 disorders x 8 samples at 128^2, chi=32, ~1 min
    python tests/golden/make_config_golden.py C4      # 1 disorder x 4 samples at 512^2, ~10 min
    python tests/golden/make_config_golden.py C5      # 1 disorder x 2 samples at 1024^2, ~40 min, ~20 GB of RAM
                                                      # (OMP_NUM_THREADS=1: the LAPACK calls are 64x128)

Per (beta, disorder) the file holds, from oracle.bmps / oracle.sampler / oracle.exact on the seeded instance
and the Philox uniforms of reading R (Eq. 1):
    logZ, logscale0                      log Z (Eq. 6) and the log-scale of row 0
    cfg_bits (n_s, L, W) uint32          sampled spins, the ABI's packing (bit c%32 of word c/32 <=> s = +1)
    logq (n_s,), E (n_s,) int64          log q(s) and the energy of every sampled configuration
    probs (n_p, len(prob_rows), L)       conditionals q(s_i = +1 | s_<i) of the first n_p samples on `prob_rows`
    min_margin (n_s,)                    min over sites of |u - p|: how close the chain came to a threshold
    floor_logZ, floor_p, floor_logq      the oracle's own rounding-noise floor (tests/noise_floor.py): the change
                                         of log Z / conditionals / log q when ONE rounding error of norm-wise noise
                                         per row is injected into the oracle's build (teacher-forced on cfg_bits)
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from oracle import bmps, exact, philox, sampler          # noqa: E402
from tnmc_workloads import CONFIGS, make_couplings        # noqa: E402
import noise_floor as nf                                  # noqa: E402
from bitpack import pack                                  # noqa: E402

# name -> (disorders, samples per disorder, samples with stored conditionals, stride of the stored rows)
SUBSETS = {
    "C2": dict(disorders=list(range(100)), n_s=32, n_p=1, row_stride=1),
    "C3": dict(disorders=[0, 255], n_s=8, n_p=2, row_stride=1),
    "C4": dict(disorders=[0], n_s=4, n_p=1, row_stride=8),
    "C5": dict(disorders=[0], n_s=2, n_p=1, row_stride=16),
}


def uniforms(seed, d, n_s, L):
    sites = np.arange(L * L)
    return philox.spin_uniforms(seed, d, np.arange(n_s)[:, None], sites[None, :]).reshape(n_s, L, L)


def build_cache_compact(Jr, Jd, beta, chi, noise_rng=None):
    """oracle.bmps.build_cache, its loop written out so that every stored row is a compact COPY:
    the tensors compress() returns are views of the 4x larger LAPACK outputs, which at L = 1024 is 68 GB instead of
    17 GB.  Same oracle calls in the same order, nothing else.  With noise_rng: tests/noise_floor.perturbed_cache
    (one rounding error of norm-wise noise per row), likewise compacted."""
    L = Jr.shape[0]
    cache = [None] * L
    logscale = np.zeros(L)
    mps = bmps.bottom_mps(Jr, beta)
    cache[L - 1] = mps
    for row in range(L - 2, -1, -1):
        mps = bmps.multiply(bmps.row_mpo(Jr, Jd, beta, row), mps)
        if noise_rng is not None:
            mps = [A + nf.EPS * np.abs(A).max() * noise_rng.standard_normal(A.shape) for A in mps]
        ls, mps, _ = bmps.compress(mps, chi)
        mps = [np.array(A) for A in mps]
        cache[row] = mps
        logscale[row] = logscale[row + 1] + ls
    return cache, logscale


def one(L, chi, beta, Jr, Jd, seed, d, n_s, n_p, prob_rows):
    compact = L >= 512
    cache, ls = build_cache_compact(Jr, Jd, beta, chi) if compact else bmps.build_cache(Jr, Jd, beta, chi)
    lz, sign = bmps.log_z(cache[0], ls[0])
    assert sign == 1.0
    u = uniforms(seed, d, n_s, L)
    cfg, logq, probs = sampler.sample(cache, Jd, beta, u)
    out = dict(logZ=lz, logscale0=ls[0], cfg_bits=pack(cfg), logq=logq, E=exact.energy(cfg, Jr, Jd),
               probs=probs[:n_p][:, prob_rows, :].copy(), min_margin=np.abs(u - probs).min(axis=(1, 2)))
    del cache
    cache_p, ls_p = (build_cache_compact(Jr, Jd, beta, chi, noise_rng=np.random.default_rng(12345)) if compact
                     else nf.perturbed_cache(Jr, Jd, beta, chi))
    lz_p, _ = bmps.log_z(cache_p[0], ls_p[0])
    fl_p, fl_q = nf.probs_floor(cache_p, Jd, beta, cfg, probs, logq)
    out.update(floor_logZ=abs(lz_p - lz), floor_p=fl_p, floor_logq=fl_q)
    return out


def main(name):
    c, s = CONFIGS[name], SUBSETS[name]
    L, chi = c["L"], c["chi"]
    prob_rows = np.arange(0, L, s["row_stride"])
    if prob_rows[-1] != L - 1:
        prob_rows = np.append(prob_rows, L - 1)
    res = {}
    t0 = time.time()
    for beta in c["betas"]:
        for d in s["disorders"]:
            Jr, Jd = make_couplings(L, 1, c["inst_seed"], first_disorder=d)
            r = one(L, chi, beta, Jr[0], Jd[0], c["seed"], d, s["n_s"], s["n_p"], prob_rows)
            for k, v in r.items():
                res.setdefault(k, []).append(v)
            print(f"{name} beta={beta} d={d}: logZ={r['logZ']:.12f} floors z={r['floor_logZ']:.2e} p={r['floor_p']:.2e} "
                  f"q={r['floor_logq']:.2e}  [{time.time() - t0:.0f} s]", flush=True)
    nb, nd = len(c["betas"]), len(s["disorders"])
    arr = {k: np.array(v).reshape((nb, nd) + np.shape(v[0])) for k, v in res.items()}
    np.savez_compressed(os.path.join(HERE, f"config_{name}.npz"), betas=np.array(c["betas"]),
                        disorders=np.array(s["disorders"]), prob_rows=prob_rows, L=L, chi=chi,
                        inst_seed=c["inst_seed"], seed=c["seed"], **arr)


if __name__ == "__main__":
    main(sys.argv[1])
