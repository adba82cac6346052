"""Pins of the oracle for real-valued couplings (Gaussian EA): Eq. 1 and the whole bMPS
path hold for any J_ij; what changes is only that energies are floats."""
import numpy as np

from oracle import bmps, exact, metropolis, sampler
from tnmc_workloads import make_couplings, make_gaussian_couplings


def test_energy_real_reduces_to_integer_energy_and_scales():
    L = 5
    Jr, Jd = make_couplings(L, 1, 3)
    rng = np.random.default_rng(0)
    cfg = rng.integers(0, 2, (7, L, L))
    assert (exact.energy_real(cfg, Jr[0], Jd[0]) == exact.energy(cfg, Jr[0], Jd[0])).all()
    assert np.allclose(exact.energy_real(cfg, 0.37 * Jr[0], 0.37 * Jd[0]), 0.37 * exact.energy(cfg, Jr[0], Jd[0]), rtol=0, atol=1e-12)
    # all-up state of a uniform ferromagnet J = 0.5: E = -0.5 * 2 L (L - 1)
    Jr1 = np.zeros((L, L)); Jr1[:, :-1] = 0.5
    Jd1 = np.zeros((L, L)); Jd1[:-1, :] = 0.5
    assert exact.energy_real(np.ones((L, L)), Jr1, Jd1) == -0.5 * 2 * L * (L - 1)


def test_single_flip_identity_gaussian():
    L = 4
    Jr, Jd = make_gaussian_couplings(L, 1, 11)
    Jr, Jd = Jr[0], Jd[0]
    rng = np.random.default_rng(1)
    cfg = rng.integers(0, 2, (L, L))
    s = 2 * cfg - 1
    E0 = exact.energy_real(cfg, Jr, Jd)
    for (r, c) in [(0, 0), (1, 2), (3, 3), (2, 0)]:
        h = 0.0
        if c + 1 < L: h += Jr[r, c] * s[r, c + 1]
        if c > 0: h += Jr[r, c - 1] * s[r, c - 1]
        if r + 1 < L: h += Jd[r, c] * s[r + 1, c]
        if r > 0: h += Jd[r - 1, c] * s[r - 1, c]
        f = cfg.copy(); f[r, c] ^= 1
        assert abs(exact.energy_real(f, Jr, Jd) - E0 - 2 * s[r, c] * h) < 1e-12


def test_exact_chi_limit_gaussian():
    """chi >= 2^(L/2): log Z = exact transfer matrix, log q(s) = -beta E(s) - log Z, every proposal accepted."""
    L, chi, beta = 6, 8, 0.9
    Jr, Jd = make_gaussian_couplings(L, 1, 5)
    Jr, Jd = Jr[0], Jd[0]
    cache, ls = bmps.build_cache(Jr, Jd, beta, chi)
    lz, sign = bmps.log_z(cache[0], ls[0])
    assert sign == 1.0 and abs(lz - exact.transfer_logZ(Jr, Jd, beta)) < 1e-10 * abs(lz)
    rng = np.random.default_rng(2)
    u = rng.random((40, L, L))
    cfg, logq, probs = sampler.sample(cache, Jd, beta, u)
    E = exact.energy_real(cfg, Jr, Jd)
    assert np.abs(logq + beta * E + lz).max() < 1e-9
    ref = exact.transfer_conditionals(Jr, Jd, beta, cfg[0])
    assert np.abs(probs[0] - ref).max() < 1e-10
    acc, n_acc, *_ = metropolis.metropolis_scan_real(E, logq, beta, rng.random(40))
    assert n_acc == 39
    # the real-energy scan reduces to the integer one on integer data
    Ei = np.array([-4, -2, -6, -4, -4]); lq = np.array([-2.0, -1.0, -3.5, -2.5, -2.5]); uu = np.array([0.0, 0.5, 0.9, 0.01, 0.999])
    a1 = metropolis.metropolis_scan(Ei, lq, 1.0, uu); a2 = metropolis.metropolis_scan_real(Ei.astype(float), lq, 1.0, uu)
    assert (a1[0] == a2[0]).all() and a1[1] == a2[1] and a1[5] == a2[5]
