"""Pins 1-4: the exact parts of the oracle against closed forms and each other."""
import math
import os

import numpy as np
import pytest

from oracle import exact
from tnmc_workloads import make_couplings

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _closed_forms():
    out = {}
    for line in open(os.path.join(GOLD, "closed_forms.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, beta, val = line.split()
        out[(name, float(beta))] = float(val)
    return out


def _ferro(L):
    Jr = np.ones((L, L), dtype=np.int8); Jr[:, L - 1] = 0
    Jd = np.ones((L, L), dtype=np.int8); Jd[L - 1, :] = 0
    return Jr, Jd


# ---- pin 1: energy, Eq. 1 -------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 3, 4, 7])
def test_energy_all_up_ferromagnet(L):
    Jr, Jd = _ferro(L)
    assert exact.energy(np.ones((L, L), dtype=np.int8), Jr, Jd) == -2 * L * (L - 1)
    assert exact.energy(np.zeros((L, L), dtype=np.int8), Jr, Jd) == -2 * L * (L - 1)


def test_energy_single_flip_and_gauge():
    L = 6
    Jr, Jd = make_couplings(L, 1, 11); Jr, Jd = Jr[0], Jd[0]
    rng = np.random.default_rng(3)
    cfg = rng.integers(0, 2, (L, L)).astype(np.int8)
    s = 2 * cfg.astype(int) - 1
    E0 = exact.energy(cfg, Jr, Jd)
    for (r, c) in [(0, 0), (2, 3), (5, 5), (0, 5), (3, 0)]:
        field = 0
        if c + 1 < L: field += Jr[r, c] * s[r, c + 1]
        if c > 0: field += Jr[r, c - 1] * s[r, c - 1]
        if r + 1 < L: field += Jd[r, c] * s[r + 1, c]
        if r > 0: field += Jd[r - 1, c] * s[r - 1, c]
        flipped = cfg.copy(); flipped[r, c] ^= 1
        assert exact.energy(flipped, Jr, Jd) - E0 == 2 * s[r, c] * field
    # gauge: J_ij -> tau_i J_ij tau_j, s -> tau s leaves E unchanged
    tau = 2 * rng.integers(0, 2, (L, L)) - 1
    Jr2 = Jr.copy(); Jd2 = Jd.copy()
    Jr2[:, :-1] = Jr[:, :-1] * tau[:, :-1] * tau[:, 1:]
    Jd2[:-1, :] = Jd[:-1, :] * tau[:-1, :] * tau[1:, :]
    cfg2 = ((s * tau + 1) // 2).astype(np.int8)
    assert exact.energy(cfg2, Jr2, Jd2) == E0


def test_energy_counts_each_bond_once():
    # one bond only: E = -J s s'
    L = 3
    Jr = np.zeros((L, L), dtype=np.int8); Jd = np.zeros((L, L), dtype=np.int8)
    Jd[1, 2] = -1
    cfg = np.zeros((L, L), dtype=np.int8); cfg[1, 2] = 1
    assert exact.energy(cfg, Jr, Jd) == -(-1) * (+1) * (-1)  # = -1
    Jr[0, 1] = 1
    assert exact.energy(cfg, Jr, Jd) == -1 - 1


# ---- pin 2: brute force and transfer matrix against closed forms ------------------------
@pytest.mark.parametrize("beta", [0.5, 1.0, 2.0])
def test_decoupled_rows_closed_form(beta):
    cf = _closed_forms()
    Jr, _ = make_couplings(4, 1, 5); Jr = Jr[0]
    Jd = np.zeros((4, 4), dtype=np.int8)
    ref = cf[("rows4x4", beta)]
    assert exact.brute_force(Jr, Jd, beta)[2] == pytest.approx(ref, rel=1e-13)
    assert exact.transfer_logZ(Jr, Jd, beta) == pytest.approx(ref, rel=1e-13)


@pytest.mark.parametrize("beta", [0.5, 1.0, 2.0])
@pytest.mark.parametrize("frustrated", [False, True])
def test_single_plaquette_closed_form(beta, frustrated):
    cf = _closed_forms()
    Jr = np.array([[1, 0], [1, 0]], dtype=np.int8)
    Jd = np.array([[1, -1 if frustrated else 1], [0, 0]], dtype=np.int8)
    ref = cf[("plaq_frustrated" if frustrated else "plaq_ferro", beta)]
    assert exact.brute_force(Jr, Jd, beta)[2] == pytest.approx(ref, rel=1e-13)
    assert exact.transfer_logZ(Jr, Jd, beta) == pytest.approx(ref, rel=1e-13)


@pytest.mark.parametrize("L", [3, 4, 8, 10])
def test_spanning_tree_closed_form(L):
    # comb: horizontal bonds on row 0 only, all vertical bonds: a tree, so
    # Z = 2^N prod_b cosh(beta J_b) whatever the signs
    Jr, Jd = make_couplings(L, 1, 21); Jr, Jd = Jr[0].copy(), Jd[0]
    Jr[1:, :] = 0
    beta = 0.8
    nb = (L - 1) + L * (L - 1)
    ref = L * L * math.log(2) + nb * math.log(math.cosh(beta))
    assert exact.transfer_logZ(Jr, Jd, beta) == pytest.approx(ref, rel=1e-13)
    if L <= 4:
        assert exact.brute_force(Jr, Jd, beta)[2] == pytest.approx(ref, rel=1e-13)


# ---- pin 3: brute force = transfer matrix on random +-J --------------------------------
@pytest.mark.parametrize("L,beta,seed", [(2, 1.0, 1), (3, 0.5, 2), (3, 2.0, 3), (4, 1.0, 4), (4, 0.3, 5)])
def test_brute_force_equals_transfer(L, beta, seed):
    Jr, Jd = make_couplings(L, 1, seed); Jr, Jd = Jr[0], Jd[0]
    cfgs, E, logZ, P = exact.brute_force(Jr, Jd, beta)
    assert P.sum() == pytest.approx(1.0, abs=1e-13)
    assert exact.transfer_logZ(Jr, Jd, beta) == pytest.approx(logZ, rel=1e-13)
    # Eq. 4 conditionals: enumeration vs transfer-matrix, along two configurations
    rng = np.random.default_rng(seed)
    for _ in range(2):
        cfg = rng.integers(0, 2, (L, L)).astype(np.int8)
        pt = exact.transfer_conditionals(Jr, Jd, beta, cfg)
        flat = cfg.reshape(-1)
        for i in range(L * L):
            pb = exact.brute_force_conditional(cfgs, P, list(flat[:i]))
            assert pt.reshape(-1)[i] == pytest.approx(pb, abs=1e-13)
        # chain rule Eq. 3: product of conditionals = Boltzmann probability
        q = np.where(flat == 1, pt.reshape(-1), 1 - pt.reshape(-1))
        e = exact.energy(cfg, Jr, Jd)
        # (1 - p loses relative precision when p -> 1 on improbable configurations: abs 1e-8)
        assert np.log(q).sum() == pytest.approx(-beta * e - logZ, abs=1e-8)


# ---- pin 4: ferromagnetic limit -----------------------------------------------------------
FERRO = {(3, 1.0): 12.809420245131097, (4, 0.5): 14.497711024011295,
         (4, 1.0): 24.817644410412711, (4, 2.0): 48.694590589829239}


@pytest.mark.parametrize("L,beta", list(FERRO))
def test_ferromagnet_logZ(L, beta):
    """Values listed in SURVEY.md 8c pin 4 (brute-force enumeration of the all-J=+1 open lattice);
    low-temperature sanity: log Z -> beta * 2L(L-1) + log 2 as beta grows."""
    Jr, Jd = _ferro(L)
    assert exact.brute_force(Jr, Jd, beta)[2] == pytest.approx(FERRO[(L, beta)], rel=1e-13)
    assert exact.transfer_logZ(Jr, Jd, beta) == pytest.approx(FERRO[(L, beta)], rel=1e-13)


def test_ferromagnet_limits_and_gauge():
    L = 10
    Jr, Jd = _ferro(L)
    # beta -> large: two ground states of energy -2L(L-1)
    beta = 6.0
    assert exact.transfer_logZ(Jr, Jd, beta) == pytest.approx(beta * 2 * L * (L - 1) + math.log(2), abs=1e-6)
    # beta = 0: Z = 2^N
    assert exact.transfer_logZ(Jr, Jd, 0.0) == pytest.approx(L * L * math.log(2), rel=1e-14)
    # any gauge transform of the ferromagnet has the same Z
    rng = np.random.default_rng(0)
    tau = 2 * rng.integers(0, 2, (L, L)) - 1
    Jr2 = Jr.copy(); Jd2 = Jd.copy()
    Jr2[:, :-1] = tau[:, :-1] * tau[:, 1:]
    Jd2[:-1, :] = tau[:-1, :] * tau[1:, :]
    assert exact.transfer_logZ(Jr2, Jd2, 1.0) == pytest.approx(exact.transfer_logZ(Jr, Jd, 1.0), rel=1e-13)
