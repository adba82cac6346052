"""Pins of oracle/potts.py (q-state Potts generalisation): the q = 2 reduction to the pinned Ising oracle,
the closed form on trees, brute force on a 3x3 q = 3 lattice, the exact-chi limit (log q = -beta E - log Z, sum of q = 1)."""
import math

import numpy as np

from oracle import bmps, exact, potts, sampler
from tnmc_workloads import make_couplings


def _exact_chi_logz(Jr, Jd, beta, q, chi):
    cache, ls = potts.build_cache(Jr, Jd, beta, chi, q)
    lz, sign = bmps.log_z(cache[0], ls[0])
    assert sign == 1.0
    return lz, cache


def test_q2_is_the_ising_model_at_half_beta():
    # delta(s,s') = (1 + sigma sigma')/2  =>  Z_potts(beta, J) = exp(beta sum_b J_b / 2) Z_ising(beta / 2, J)
    L, beta = 5, 1.3
    Jr, Jd = make_couplings(L, 1, 91)
    Jr, Jd = Jr[0].astype(float), Jd[0].astype(float)
    lz_p, cache_p = _exact_chi_logz(Jr, Jd, beta, 2, 16)
    lz_i = exact.transfer_logZ(Jr, Jd, beta / 2.0)
    assert abs(lz_p - (beta * (Jr.sum() + Jd.sum()) / 2.0 + lz_i)) < 1e-10 * abs(lz_p)
    # and the conditionals: Potts p(s = 1 | s_<i) = Ising q(s = +1 | s_<i) at beta / 2, site by site
    rng = np.random.default_rng(3)
    u = rng.random((6, L, L))
    cfg_p, logq_p, probs_p = potts.sample(cache_p, Jd, beta, u, 2)
    cache_i, _ = bmps.build_cache(Jr, Jd, beta / 2.0, 16)
    cfg_i, logq_i, probs_i = sampler.sample(cache_i, Jd, beta / 2.0, np.zeros_like(u), forced=cfg_p)
    assert np.abs(probs_p[..., 1] - probs_i).max() < 1e-10
    assert np.abs(logq_p - logq_i).max() < 1e-9


def test_tree_closed_form():
    # bonds forming a tree (a comb: the first column and every row): Z = q^N prod_b (e^{beta J_b} + q - 1) / q
    L, beta, q = 4, 0.7, 3
    rng = np.random.default_rng(8)
    Jr = np.zeros((L, L)); Jd = np.zeros((L, L))
    Jr[:, : L - 1] = rng.choice([-1.0, 1.0, 0.5], size=(L, L - 1))
    Jd[: L - 1, 0] = rng.choice([-1.0, 1.0], size=L - 1)
    bonds = list(Jr[:, : L - 1].ravel()) + list(Jd[: L - 1, 0])
    lz_exact = L * L * math.log(q) + sum(math.log((math.exp(beta * J) + q - 1) / q) for J in bonds)
    lz, _ = _exact_chi_logz(Jr, Jd, beta, q, 81)
    assert abs(lz - lz_exact) < 1e-10 * abs(lz_exact)


def test_3x3_q3_brute_force_and_exact_chi_sampling():
    L, beta, q = 3, 0.9, 3
    Jr, Jd = make_couplings(L, 1, 92)
    Jr, Jd = Jr[0].astype(float), Jd[0].astype(float)
    cfgs, E, logZ, P = potts.brute_force(Jr, Jd, beta, q)
    assert len(cfgs) == q ** (L * L) and abs(P.sum() - 1.0) < 1e-12
    lz, cache = _exact_chi_logz(Jr, Jd, beta, q, 27)
    assert abs(lz - logZ) < 1e-10 * abs(logZ)
    # teacher-forced over ALL configurations: exp(log q) is the Boltzmann distribution, so sum q = 1 and
    # log q = -beta E - log Z configuration by configuration
    _, logq, probs = potts.sample(cache, Jd, beta, np.zeros((len(cfgs), L, L)), q, forced=cfgs)
    assert np.abs(logq - (-beta * E - logZ)).max() < 1e-9
    assert abs(np.exp(logq).sum() - 1.0) < 1e-10
    assert np.abs(probs.sum(axis=-1) - 1.0).max() < 1e-12
    # free sampling: the categorical draw picks the outcome whose cumulative interval holds u
    rng = np.random.default_rng(5)
    u = rng.random((2000, L, L))
    cfg, lq, pr = potts.sample(cache, Jd, beta, u, q)
    cum = np.cumsum(pr, axis=-1)
    lo = np.concatenate([np.zeros(pr.shape[:-1] + (1,)), cum[..., :-1]], axis=-1)
    pick = np.take_along_axis(lo, cfg[..., None].astype(np.int64), axis=-1)[..., 0]
    top = np.take_along_axis(cum, cfg[..., None].astype(np.int64), axis=-1)[..., 0]
    assert ((pick <= u) & ((u < top) | (cfg == q - 1))).all()
    # histogram of the 2000 exact samples against the Boltzmann probabilities (chi-square over the 30 likeliest states)
    idx = (cfg.reshape(len(cfg), -1).astype(np.int64) * (q ** np.arange(L * L - 1, -1, -1))).sum(axis=1)
    counts = np.bincount(idx, minlength=len(cfgs))
    top30 = np.argsort(-P)[:30]
    chi2 = (((counts[top30] - 2000 * P[top30]) ** 2) / (2000 * P[top30])).sum()
    assert chi2 < 70.0                                   # 30 cells: mean 30, 5-sigma ~ 69


def test_truncated_potts_is_a_normalised_sampler():
    # chi below the exact bound: q(s) is still a normalised distribution and close to Boltzmann
    L, beta, q = 3, 0.6, 3
    Jr, Jd = make_couplings(L, 1, 93)
    Jr, Jd = Jr[0].astype(float), Jd[0].astype(float)
    cfgs, E, logZ, P = potts.brute_force(Jr, Jd, beta, q)
    cache, ls = potts.build_cache(Jr, Jd, beta, 5, q)
    _, logq, _ = potts.sample(cache, Jd, beta, np.zeros((len(cfgs), L, L)), q, forced=cfgs)
    assert abs(np.exp(logq).sum() - 1.0) < 1e-10
    assert 0.5 * np.abs(np.exp(logq) - P).sum() < 0.05
