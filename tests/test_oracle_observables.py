"""Pins of oracle/observables.py: a hand-worked chain, the all-up / all-down magnetisation, and the
exact-chi limit, where the chain is an exact Boltzmann sampler and its averages must converge to the
brute-force thermal averages (statistical, 4-sigma bands)."""
import numpy as np

from oracle import bmps, exact, metropolis, observables, philox, sampler
from tnmc_workloads import make_couplings


def test_magnetisation_definition():
    L = 5
    up = np.ones((L, L), dtype=np.int8)
    assert observables.magnetisation(up) == L * L
    assert observables.magnetisation(1 - up) == -L * L
    c = up.copy(); c[2, 3] = 0
    assert observables.magnetisation(c) == L * L - 2
    assert (observables.magnetisation(np.stack([up, c])) == [25, 23]).all()


def test_chain_sums_hand_worked():
    # the chain of tests/golden/metropolis_hand.txt: flags 1 0 1 1 1, energies -4 -2 -6 -4 -4; M chosen here
    E = [-4, -2, -6, -4, -4]
    M = [2, 0, -4, 6, 2]
    acc = [1, 0, 1, 1, 1]
    # states visited: (-4,2) (-4,2) (-6,-4) (-4,6) (-4,2)
    s, cE, cM = observables.chain_sums(E, M, acc)
    assert s == [-22, 16 + 16 + 36 + 16 + 16, 8, 16, 4 + 4 + 16 + 36 + 4]
    assert (cE, cM) == (-4, 2)
    # chunked: same sums, state carried
    s1, cE, cM = observables.chain_sums(E[:2], M[:2], acc[:2])
    s2, cE, cM = observables.chain_sums(E[2:], M[2:], acc[2:], cE, cM)
    assert [a + b for a, b in zip(s1, s2)] == s
    # a chunk that starts with a rejection stays on the carried state
    s3, _, _ = observables.chain_sums([5], [9], [0], cur_E=-6, cur_M=-4)
    assert s3 == [-6, 36, -4, 4, 16]


def test_chain_sums_real_reduces_to_integer_version():
    E = [-4, -2, -6, -4, -4]; M = [2, 0, -4, 6, 2]; acc = [1, 0, 1, 1, 1]
    s, cE, cM = observables.chain_sums(E, M, acc)
    sr, cEr, cMr = observables.chain_sums_real([float(e) for e in E], M, acc)
    assert sr == [float(s[0]), float(s[1]), s[2], s[3], s[4]] and (cEr, cMr) == (float(cE), cM)
    sh, _, _ = observables.chain_sums_real([0.5, -1.25], [1, -3], [1, 1])
    assert sh == [-0.75, 0.25 + 1.5625, -2, 4, 10]


def test_exact_chi_chain_reproduces_boltzmann_averages():
    L, chi, beta, n_s, seed = 3, 8, 0.8, 6000, 21
    Jr, Jd = make_couplings(L, 1, 77)
    Jr, Jd = Jr[0], Jd[0]
    cfgs, E_all, logZ, Pb = exact.brute_force(Jr, Jd, beta)
    M_all = observables.magnetisation(cfgs)
    cache, _ = bmps.build_cache(Jr, Jd, beta, chi)
    u = np.empty((n_s, L, L))
    for r in range(L):
        for c in range(L):
            u[:, r, c] = philox.spin_uniforms(seed, 0, np.arange(n_s), r * L + c)
    cfg, logq, _ = sampler.sample(cache, Jd, beta, u)
    E = exact.energy(cfg, Jr, Jd)
    M = observables.magnetisation(cfg)
    um = philox.metropolis_uniforms(seed, 0, np.arange(n_s))
    acc, n_acc, *_ = metropolis.metropolis_scan(E, logq, beta, um)
    assert n_acc >= n_s - 3                      # exact chi: (almost) every proposal is accepted
    s, _, _ = observables.chain_sums(E, M, acc)
    for est, exact_val, exact_sq in ((s[0] / n_s, (Pb * E_all).sum(), (Pb * E_all ** 2).sum()),
                                     (s[3] / n_s, (Pb * np.abs(M_all)).sum(), (Pb * M_all ** 2).sum()),
                                     (s[4] / n_s, (Pb * M_all ** 2).sum(), (Pb * M_all.astype(float) ** 4).sum())):
        sigma = np.sqrt(max(exact_sq - exact_val ** 2, 1e-12) / n_s)
        assert abs(est - exact_val) < 4.5 * sigma
