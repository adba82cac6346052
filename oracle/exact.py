"""Oracle Part E: exact definitions, small lattices only (test infrastructure).

E1  energy, Eq. 1:   E(s) = - sum_<ij> J_ij s_i s_j
E2  brute force over all 2^N states: Z (Eq. 6), Boltzmann P(s) (Eq. 2,
    PAPER.md:53, printed "1/7" = 1/Z), conditionals by Eq. 4.
E3  exact row-transfer-matrix state vectors: the textbook restatement of contracting
    Fig. 1(b) one row at a time, bottom to top, with the boundary held as
    a full 2^L vector instead of an MPS.  Psi_r(sigma) = sum over all spins in rows > r
    of the Boltzmann weight of every bond inside rows r..L-1, row r clamped to sigma.

Layout: Jr[r,c] couples (r,c)-(r,c+1) (0 at c=L-1); Jd[r,c] couples (r,c)-(r+1,c)
(0 at r=L-1).  Spin index a in {0,1} <-> s = 2a-1.  Raster order site = r*L + c
(PAPER.md:60).  A row configuration sigma is an integer whose bit c is a_c.
"""
import itertools
import numpy as np


def energy(cfg, Jr, Jd):
    """E1. cfg: (..., L, L) array of {0,1}; returns integer energy, Eq. 1."""
    s = 2 * np.asarray(cfg, dtype=np.int64) - 1
    Jr = np.asarray(Jr, dtype=np.int64)
    Jd = np.asarray(Jd, dtype=np.int64)
    e_right = (s[..., :, :-1] * s[..., :, 1:] * Jr[:, :-1]).sum(axis=(-1, -2))
    e_down = (s[..., :-1, :] * s[..., 1:, :] * Jd[:-1, :]).sum(axis=(-1, -2))
    return -(e_right + e_down)


def energy_real(cfg, Jr, Jd):
    """E1 for real-valued couplings (Eq. 1 holds for any J_ij): float64."""
    s = 2.0 * np.asarray(cfg, dtype=np.float64) - 1.0
    Jr = np.asarray(Jr, dtype=np.float64)
    Jd = np.asarray(Jd, dtype=np.float64)
    e_right = (s[..., :, :-1] * s[..., :, 1:] * Jr[:, :-1]).sum(axis=(-1, -2))
    e_down = (s[..., :-1, :] * s[..., 1:, :] * Jd[:-1, :]).sum(axis=(-1, -2))
    return -(e_right + e_down)


def all_configs(L):
    """(2^(L*L), L, L) array of every configuration, raster bit order (site 0 = MSB)."""
    n = L * L
    return np.array(list(itertools.product((0, 1), repeat=n)), dtype=np.int8).reshape(-1, L, L)


def brute_force(Jr, Jd, beta):
    """E2. Returns (cfgs, energies, logZ, P) by enumeration.  N = L*L <= ~20."""
    L = Jr.shape[0]
    cfgs = all_configs(L)
    E = energy(cfgs, Jr, Jd)
    w = -beta * E.astype(np.float64)
    m = w.max()
    logZ = m + np.log(np.exp(w - m).sum())
    return cfgs, E, logZ, np.exp(w - logZ)


def brute_force_conditional(cfgs, P, prefix):
    """Eq. 4: P(s_i = +1 | s_<i) with i = len(prefix), from the enumerated Boltzmann P."""
    n = cfgs.shape[0]
    flat = cfgs.reshape(n, -1)
    i = len(prefix)
    sel = np.ones(n, dtype=bool)
    for k, a in enumerate(prefix):
        sel &= flat[:, k] == a
    den = P[sel].sum()
    num = P[sel & (flat[:, i] == 1)].sum()
    return num / den


def bmat(beta, J):
    """Eq. 7: B[a,b] = exp(beta*J*(2a-1)(2b-1))."""
    s = np.array([-1.0, 1.0])
    return np.exp(beta * float(J) * np.outer(s, s))


def _apply_on_axis(vec, mat, L, c):
    """vec'(.., a_c=x, ..) = sum_y mat[x,y] vec(.., a_c=y, ..); bit c of the index is a_c."""
    t = vec.reshape([2] * L)           # axis k <-> bit (L-1-k) in C order
    ax = L - 1 - c
    t = np.moveaxis(np.tensordot(mat, t, axes=([1], [ax])), 0, ax)
    return t.reshape(-1)


def _row_weight(beta, Jr_row, L):
    """prod_c B(Jr[c])[a_c, a_{c+1}] for every row configuration (length 2^L)."""
    idx = np.arange(1 << L)
    a = ((idx[:, None] >> np.arange(L)[None, :]) & 1).astype(np.float64)   # a[:, c]
    s = 2 * a - 1
    expo = (s[:, :-1] * s[:, 1:] * np.asarray(Jr_row[:-1], dtype=np.float64)).sum(axis=1)
    return np.exp(beta * expo)


def transfer_states(Jr, Jd, beta):
    """E3. list over r of (vec_r, log_r) with Psi_r = exp(log_r) * vec_r, |vec_r|_2 = 1."""
    L = Jr.shape[0]
    out = [None] * L
    v = _row_weight(beta, Jr[L - 1], L)
    lg = 0.0
    nrm = np.linalg.norm(v); v = v / nrm; lg += np.log(nrm)
    out[L - 1] = (v, lg)
    for r in range(L - 2, -1, -1):
        for c in range(L):
            v = _apply_on_axis(v, bmat(beta, Jd[r, c]), L, c)    # sum over the row below
        v = v * _row_weight(beta, Jr[r], L)
        nrm = np.linalg.norm(v); v = v / nrm; lg += np.log(nrm)
        out[r] = (v, lg)
    return out


def transfer_logZ(Jr, Jd, beta):
    v, lg = transfer_states(Jr, Jd, beta)[0]
    return lg + np.log(v.sum())


def transfer_conditionals(Jr, Jd, beta, cfg, states=None):
    """Exact P(s_{r,c}=+1 | s_<(r,c)) for every site of one configuration cfg (L,L) by Eq. 4,
    using f(s_i, s_<i) ~ sum_{sigma: sigma_<c fixed, sigma_c = a} prod_c' B(Ju)[up_c', sigma_c'] Psi_r(sigma)
    (the weights of bonds between already-fixed spins cancel in the ratio)."""
    L = Jr.shape[0]
    if states is None:
        states = transfer_states(Jr, Jd, beta)
    idx = np.arange(1 << L)
    bits = (idx[:, None] >> np.arange(L)[None, :]) & 1
    probs = np.zeros((L, L))
    for r in range(L):
        v = states[r][0].copy()
        if r > 0:
            for c in range(L):
                su = 2.0 * cfg[r - 1, c] - 1.0
                v = v * np.exp(beta * float(Jd[r - 1, c]) * su * (2.0 * bits[:, c] - 1.0))
        sel = np.ones(1 << L, dtype=bool)
        for c in range(L):
            f1 = v[sel & (bits[:, c] == 1)].sum()
            f0 = v[sel & (bits[:, c] == 0)].sum()
            probs[r, c] = f1 / (f0 + f1)
            sel &= bits[:, c] == cfg[r, c]
    return probs
