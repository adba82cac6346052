"""Pins 5-7: the bMPS build and the sampler of the oracle."""
import numpy as np
import pytest

from oracle import bmps, exact, sampler
from tnmc_workloads import make_couplings


def _inst(L, seed):
    Jr, Jd = make_couplings(L, 1, seed)
    return Jr[0], Jd[0]


def test_shapes_follow_paper():
    """MPS [(1,2,chi),(chi,2,chi),...,(chi,2,1)], MPO [(1,2,2,2),(2,2,2,2),...,(2,2,1,2)]."""
    L, chi = 8, 4
    Jr, Jd = _inst(L, 1)
    mpo = bmps.row_mpo(Jr, Jd, 1.0, 3)
    assert [W.shape for W in mpo] == [(1, 2, 2, 2)] + [(2, 2, 2, 2)] * (L - 2) + [(2, 2, 1, 2)]
    bot = bmps.bottom_mps(Jr, 1.0)
    assert [A.shape for A in bot] == [(1, 2, 2)] + [(2, 2, 2)] * (L - 2) + [(2, 2, 1)]
    cache, _ = bmps.build_cache(Jr, Jd, 1.0, chi)
    # interior bonds of the top rows are saturated at chi
    assert [A.shape for A in cache[0]] == [(1, 2, 2), (2, 2, 4)] + [(4, 2, 4)] * (L - 4) + [(4, 2, 2), (2, 2, 1)]


def test_mpo_and_bottom_row_elements():
    """Eq. 7/8 element by element: W[l,a,r,d] = delta(l,a) B_r[a,r] B_d[a,d]."""
    Jr, Jd = _inst(5, 2)
    beta = 0.7
    row = 1
    mpo = bmps.row_mpo(Jr, Jd, beta, row)
    s = [-1.0, 1.0]
    for c, W in enumerate(mpo):
        for l in range(W.shape[0]):
            for a in range(2):
                for r in range(W.shape[2]):
                    for d in range(2):
                        br = np.exp(beta * Jr[row, c] * s[a] * s[r]) if c < 4 else 1.0
                        bd = np.exp(beta * Jd[row, c] * s[a] * s[d])
                        delta = 1.0 if (c == 0 or l == a) else 0.0
                        assert W[l, a, r, d] == pytest.approx(delta * br * bd, rel=1e-15)


@pytest.mark.parametrize("L,chi,beta,seed", [(4, 4, 1.0, 1), (6, 8, 0.5, 2), (8, 16, 1.0, 3), (8, 16, 2.0, 4), (5, 8, 1.0, 5)])
def test_exact_chi_limit(L, chi, beta, seed):
    """Pin 5 (north_star): chi >= 2^(L/2) makes the bMPS exact: every cached row equals the exact
    transfer-matrix state, log Z is exact, every conditional equals Eq. 4, log q = -beta E - log Z."""
    Jr, Jd = _inst(L, seed)
    cache, ls = bmps.build_cache(Jr, Jd, beta, chi)
    states = exact.transfer_states(Jr, Jd, beta)
    for r in range(L):
        v = bmps.mps_to_vector(cache[r])
        nv = np.linalg.norm(v)
        assert np.abs(v / nv - states[r][0]).max() < 1e-12
        assert ls[r] + np.log(nv) == pytest.approx(states[r][1], rel=1e-13)
    logZ, sign = bmps.log_z(cache[0], ls[0])
    assert sign == 1.0
    logZ_exact = exact.transfer_logZ(Jr, Jd, beta)
    assert logZ == pytest.approx(logZ_exact, rel=1e-13)
    rng = np.random.default_rng(seed)
    u = rng.random((32, L, L))
    cfgs, logq, probs = sampler.sample(cache, Jd, beta, u)
    E = exact.energy(cfgs, Jr, Jd)
    assert np.abs(logq - (-beta * E - logZ_exact)).max() < 1e-10
    for n in range(4):
        pe = exact.transfer_conditionals(Jr, Jd, beta, cfgs[n], states)
        assert np.abs(pe - probs[n]).max() < 1e-11


def test_exact_chi_4x4_brute_force():
    """BASELINE configs[0]: 4x4 brute-force check: sampled log q = log of the enumerated Boltzmann P."""
    Jr, Jd = _inst(4, 9)
    beta = 1.0
    cfgs_all, E_all, logZ, P = exact.brute_force(Jr, Jd, beta)
    cache, ls = bmps.build_cache(Jr, Jd, beta, 4)
    assert bmps.log_z(cache[0], ls[0])[0] == pytest.approx(logZ, rel=1e-13)
    # teacher-force every one of the 65536 configurations
    _, logq, _ = sampler.sample(cache, Jd, beta, np.zeros((1 << 16, 4, 4)), forced=cfgs_all)
    assert np.abs(np.exp(logq) - P).max() < 1e-13
    assert np.exp(logq).sum() == pytest.approx(1.0, abs=1e-12)


def test_multiply_matches_exact_row_application():
    """MPO x MPS (Fig. 2) at bond dimension 2 -> 4 equals one exact transfer-matrix step."""
    L = 6
    Jr, Jd = _inst(L, 7)
    beta = 1.0
    states = exact.transfer_states(Jr, Jd, beta)
    mps = bmps.multiply(bmps.row_mpo(Jr, Jd, beta, L - 2), bmps.bottom_mps(Jr, beta))
    assert [A.shape for A in mps] == [(1, 2, 4)] + [(4, 2, 4)] * (L - 2) + [(4, 2, 1)]
    v = bmps.mps_to_vector(mps)
    assert np.abs(v / np.linalg.norm(v) - states[L - 2][0]).max() < 1e-13


@pytest.mark.parametrize("chi", [2, 3, 4])
def test_compress_eckart_young_and_canonical_form(chi):
    """Pin 6: the truncation errors of the right-to-left sweep are mutually orthogonal, so
    |Psi - Psi_trunc|^2 = sum of the discarded squared singular values; the kept tensors
    are right-isometries and the state has unit norm."""
    L = 8
    Jr, Jd = _inst(L, 13)
    beta = 1.0
    mps = bmps.bottom_mps(Jr, beta)
    for row in (L - 2, L - 3, L - 4):
        mps = bmps.multiply(bmps.row_mpo(Jr, Jd, beta, row), mps)
    before = bmps.mps_to_vector(mps)
    ls, out, disc = bmps.compress(mps, chi)
    after = bmps.mps_to_vector(out)
    assert np.linalg.norm(after) == pytest.approx(1.0, abs=1e-13)
    # exp(ls) * after is the truncated state; before/|before| the exact one
    nb = np.linalg.norm(before)
    err2 = np.linalg.norm(before / nb - np.exp(ls) * after / nb) ** 2
    assert err2 == pytest.approx(disc.sum(), rel=1e-9, abs=1e-28)
    assert disc.sum() > 0
    for A in out[1:]:
        M = A.reshape(A.shape[0], -1)
        assert np.abs(M @ M.T - np.eye(M.shape[0])).max() < 1e-13
    assert max(A.shape[0] for A in out) <= chi
    # exact when chi is large enough
    ls2, out2, disc2 = bmps.compress(mps, 64)
    assert np.abs(before - np.exp(ls2) * bmps.mps_to_vector(out2)).max() < 1e-12 * nb
    assert disc2.sum() < 1e-28


def test_qr_svd_library_steps_against_scipy():
    """The library steps themselves: numpy.linalg.qr / svd vs scipy.linalg on random matrices."""
    import scipy.linalg as sla
    rng = np.random.default_rng(0)
    M = rng.standard_normal((24, 12))
    Q, R = np.linalg.qr(M)
    Q2, R2 = sla.qr(M, mode="economic")
    sg = np.sign(np.diag(R)) * np.sign(np.diag(R2))
    assert np.abs(Q * sg - Q2).max() < 1e-13 and np.abs(R * sg[:, None] - R2).max() < 1e-13
    assert np.abs(np.linalg.svd(M, compute_uv=False) - sla.svdvals(M)).max() < 1e-13


@pytest.mark.parametrize("L,chi", [(3, 1), (4, 2), (4, 3)])
def test_truncated_q_is_normalised(L, chi):
    """Pin 7: under truncation q is still an exact autoregressive distribution: sum_s q(s) = 1."""
    Jr, Jd = _inst(L, 17)
    beta = 1.0
    cache, _ = bmps.build_cache(Jr, Jd, beta, chi)
    allc = exact.all_configs(L)
    _, logq, probs = sampler.sample(cache, Jd, beta, np.zeros((allc.shape[0], L, L)), forced=allc)
    assert np.exp(logq).sum() == pytest.approx(1.0, abs=1e-12)
    assert (probs > 0).all() and (probs < 1).all()
    # and it is NOT the Boltzmann distribution (the truncation bites)
    _, E, logZ, P = exact.brute_force(Jr, Jd, beta)
    assert np.abs(np.exp(logq) - P).max() > 1e-8


def test_gauge_covariance_under_truncation():
    """Pin 7: J -> tau J tau, s -> tau s: singular values are gauge invariant, so truncated
    log Z is unchanged and q_J'(tau s) = q_J(s)."""
    L, chi, beta = 6, 3, 1.0
    Jr, Jd = _inst(L, 23)
    rng = np.random.default_rng(1)
    tau = 2 * rng.integers(0, 2, (L, L)) - 1
    Jr2 = Jr.copy(); Jd2 = Jd.copy()
    Jr2[:, :-1] = Jr[:, :-1] * tau[:, :-1] * tau[:, 1:]
    Jd2[:-1, :] = Jd[:-1, :] * tau[:-1, :] * tau[1:, :]
    c1, l1 = bmps.build_cache(Jr, Jd, beta, chi)
    c2, l2 = bmps.build_cache(Jr2, Jd2, beta, chi)
    assert bmps.log_z(c2[0], l2[0])[0] == pytest.approx(bmps.log_z(c1[0], l1[0])[0], rel=1e-12)
    cfg = rng.integers(0, 2, (16, L, L)).astype(np.int8)
    cfg2 = (((2 * cfg - 1) * tau + 1) // 2).astype(np.int8)
    z = np.zeros((16, L, L))
    q1 = sampler.sample(c1, Jd, beta, z, forced=cfg)[1]
    q2 = sampler.sample(c2, Jd2, beta, z, forced=cfg2)[1]
    assert np.abs(q1 - q2).max() < 1e-10


def test_logZ_error_shrinks_with_chi():
    L, beta = 8, 1.0
    Jr, Jd = _inst(L, 29)
    ref = exact.transfer_logZ(Jr, Jd, beta)
    err = []
    for chi in (2, 4, 8, 16):
        cache, ls = bmps.build_cache(Jr, Jd, beta, chi)
        err.append(abs(bmps.log_z(cache[0], ls[0])[0] - ref))
    assert err[3] < 1e-11
    assert err[0] > err[2] > err[3]
    assert err[0] > 1e-6


def test_draw_semantics():
    """spin up iff u < p: u = 0 gives all up, u -> 1 gives all down."""
    L = 5
    Jr, Jd = _inst(L, 31)
    cache, _ = bmps.build_cache(Jr, Jd, 1.0, 4)
    up, lq_up, _ = sampler.sample(cache, Jd, 1.0, np.zeros((2, L, L)))
    dn, lq_dn, _ = sampler.sample(cache, Jd, 1.0, np.full((2, L, L), 1.0 - 2.0 ** -53))
    assert (up == 1).all() and (dn == 0).all()
    # zero field: q is symmetric under the global flip
    assert lq_up[0] == pytest.approx(lq_dn[0], abs=1e-10)


def test_sampler_statistics_match_boltzmann_3x3():
    """Exact chi on 3x3: the empirical histogram of 40000 draws matches Boltzmann (chi-square)."""
    from oracle import philox
    L, beta = 3, 0.6
    Jr, Jd = _inst(L, 37)
    cache, _ = bmps.build_cache(Jr, Jd, beta, 2)
    n = 40000
    u = np.zeros((n, L, L))
    for r in range(L):
        for c in range(L):
            u[:, r, c] = philox.spin_uniforms(12345, 0, np.arange(n), r * L + c)
    cfgs, _, _ = sampler.sample(cache, Jd, beta, u)
    _, _, _, P = exact.brute_force(Jr, Jd, beta)
    code = (cfgs.reshape(n, -1) * (1 << np.arange(L * L - 1, -1, -1))).sum(axis=1)
    counts = np.bincount(code, minlength=1 << (L * L))
    chi2 = ((counts - n * P) ** 2 / (n * P)).sum()
    dof = (1 << (L * L)) - 1
    assert abs(chi2 - dof) < 6 * np.sqrt(2 * dof)
