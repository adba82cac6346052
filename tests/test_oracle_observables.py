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


def test_overlap_definition_and_hand_worked_chain():
    L = 3
    up = np.ones((L, L), dtype=np.int8)
    assert observables.overlap(up, up) == 9 and observables.overlap(up, 1 - up) == -9
    c = up.copy(); c[0, 1] = 0; c[2, 2] = 0                      # differs from `up` on two sites
    assert observables.overlap(up, c) == 9 - 4 and observables.overlap(c, up) == 5
    assert observables.overlap(c, c) == 9
    d = up.copy(); d[0, 1] = 0; d[1, 1] = 0                      # c and d differ on (2,2) and (1,1)
    assert observables.overlap(c, d) == 9 - 4
    # two chains, worked by hand: chain a proposals (up, c, d), flags 1 0 1 -> states up, up, d
    #                             chain b proposals (c, c, up), flags 1 1 0 -> states c, c, c
    q, s, ca, cb = observables.replica_overlap([up, c, d], [1, 0, 1], [c, c, up], [1, 1, 0])
    assert list(q) == [5, 5, 5] and s == [15, 15, 75]            # up.c = 5, up.c = 5, d.c = 5
    assert (ca == d).all() and (cb == c).all()
    q, s, _, _ = observables.replica_overlap([up, 1 - up, c], [1, 1, 1], [up, up, 1 - c], [1, 0, 1])
    assert list(q) == [9, -9, -9] and s == [-9, 27, 243]
    # chunked with carried states = whole; a chunk starting on a rejection uses the carried state
    q1, s1, ca, cb = observables.replica_overlap([up, 1 - up], [1, 1], [up, up], [1, 0])
    q2, s2, ca, cb = observables.replica_overlap([c], [1], [1 - c], [1], ca, cb)
    assert list(q1) + list(q2) == list(q) and [x + y for x, y in zip(s1, s2)] == s
    q3, s3, _, _ = observables.replica_overlap([c], [0], [c], [0], cur_a=up, cur_b=1 - up)
    assert list(q3) == [-9] and s3 == [-9, 9, 81]


def test_overlap_symmetries():
    rng = np.random.default_rng(5)
    a = rng.integers(0, 2, size=(7, 6, 6)); b = rng.integers(0, 2, size=(7, 6, 6))
    q = observables.overlap(a, b)
    assert (q == observables.overlap(b, a)).all()                              # symmetric
    assert (observables.overlap(1 - a, b) == -q).all()                         # global flip of one replica
    assert (observables.overlap(1 - a, 1 - b) == q).all()                      # Z2 symmetry of the pair
    assert (q == 36 - 2 * (a != b).sum(axis=(1, 2))).all()                     # N - 2 Hamming distance
    assert (np.abs(q) <= 36).all() and ((q - 36) % 2 == 0).all()


def test_exact_chi_replicas_reproduce_boltzmann_overlap():
    """two independent exact samplers of the same disorder: <q^2> -> sum_{s,s'} P(s) P(s') (s.s')^2 (brute force)"""
    L, chi, beta, n_s = 3, 8, 0.9, 5000
    Jr, Jd = make_couplings(L, 1, 78)
    Jr, Jd = Jr[0], Jd[0]
    cfgs, E_all, logZ, Pb = exact.brute_force(Jr, Jd, beta)
    S = (2 * cfgs.reshape(len(cfgs), -1).astype(np.int64) - 1)
    Q = S @ S.T
    q2_exact = float(Pb @ (Q ** 2) @ Pb)
    q4_exact = float(Pb @ (Q.astype(float) ** 4) @ Pb)
    cache, _ = bmps.build_cache(Jr, Jd, beta, chi)
    chains = []
    for seed in (31, 32):
        u = np.empty((n_s, L, L))
        for r in range(L):
            for c in range(L):
                u[:, r, c] = philox.spin_uniforms(seed, 0, np.arange(n_s), r * L + c)
        cfg, logq, _ = sampler.sample(cache, Jd, beta, u)
        E = exact.energy(cfg, Jr, Jd)
        acc, n_acc, *_ = metropolis.metropolis_scan(E, logq, beta, philox.metropolis_uniforms(seed, 0, np.arange(n_s)))
        assert n_acc >= n_s - 3
        chains.append((cfg, acc))
    q, s, _, _ = observables.replica_overlap(chains[0][0], chains[0][1], chains[1][0], chains[1][1])
    sigma = np.sqrt(max(q4_exact - q2_exact ** 2, 1e-12) / n_s)
    assert abs(s[2] / n_s - q2_exact) < 4.5 * sigma
    assert abs(s[0] / n_s) < 4.5 * np.sqrt(q2_exact / n_s)                     # <q> = 0 by the Z2 symmetry
