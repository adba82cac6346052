"""Oracle, q-state Potts generalisation (test infrastructure, see oracle/__init__.py).

PAPER.md:307 names "the q-state Potts [model]" as the generalisation of the package; the paper shows no
code for it.  This module restates the method of PAPER.md:84-91 (Eq. 7-8), :150-189 (boundary-MPS cache) and
:202-254 (row-by-row ancestral sampling) with the physical dimension 2 replaced by q:
    E(s) = - sum_<ij> J_ij delta(s_i, s_j),   s_i in {0, ..., q-1}      (the Potts convention; reading G20)
    Boltzmann matrix  B[a,b] = exp(beta J delta(a,b))                    (Eq. 7 with delta in place of s s')
    copy tensors of dimension q                                          (Eq. 8)
`multiply`, `compress` and `log_z` of oracle/bmps.py take the physical dimension from the tensor shapes and are used
as they stand.  For q = 2, delta(s,s') = (1 + sigma sigma')/2, so the model IS the Ising model at beta/2 up to a
constant:  Z_potts(beta, J) = exp(beta sum_b J_b / 2) Z_ising(beta/2, J)  -- the first pin of tests/test_oracle_potts.py.
The categorical draw uses one uniform per site: s = #{a : cumulative p_a <= u} (for q = 2: s = 0 iff u < p_0).
Status: oracle only -- no CUDA kernel consumes q > 2 yet.
"""
import itertools

import numpy as np

from . import bmps


def potts_bmat(beta, J, q):
    return np.exp(beta * float(J) * np.eye(q))


def copy_tensors(q):
    I2 = np.eye(q)
    I3 = np.zeros((q, q, q))
    I4 = np.zeros((q, q, q, q))
    for i in range(q):
        I3[i, i, i] = 1.0
        I4[i, i, i, i] = 1.0
    return I2, I3, I4


def bottom_mps(Jr, beta, q):
    """PAPER.md:157-163 with dimension q: shapes [(1,q,q), (q,q,q) ..., (q,q,1)]."""
    L = Jr.shape[0]
    I2, I3, _ = copy_tensors(q)
    mps = [(I2 @ potts_bmat(beta, Jr[L - 1, 0], q))[None, :, :]]
    for col in range(1, L - 1):
        mps.append(I3 @ potts_bmat(beta, Jr[L - 1, col], q))
    mps.append(I2[:, :, None])
    return mps


def row_mpo(Jr, Jd, beta, row, q):
    """PAPER.md:169-182 with dimension q (interior line: reading G4)."""
    L = Jr.shape[0]
    _, I3, I4 = copy_tensors(q)
    B = lambda J: potts_bmat(beta, J, q)
    mpo = [np.einsum("ijk,jl,km->ilm", I3, B(Jr[row, 0]), B(Jd[row, 0]))[None]]
    for col in range(1, L - 1):
        mpo.append(np.einsum("laxy,xr,yd->lard", I4, B(Jr[row, col]), B(Jd[row, col])))
    mpo.append(np.einsum("ijk,kl->ijl", I3, B(Jd[row, L - 1]))[:, :, None, :])
    return mpo


def build_cache(Jr, Jd, beta, chi, q):
    """create_cache for the Potts model: (cache, logscale) as oracle.bmps.build_cache."""
    L = Jr.shape[0]
    cache = [None] * L
    logscale = np.zeros(L)
    mps = bottom_mps(Jr, beta, q)
    cache[L - 1] = mps
    for row in range(L - 2, -1, -1):
        mps = bmps.multiply(row_mpo(Jr, Jd, beta, row, q), mps)
        ls, mps, _ = bmps.compress(mps, chi)
        cache[row] = mps
        logscale[row] = logscale[row + 1] + ls
    return cache, logscale


def energy(cfg, Jr, Jd):
    """E = - sum_<ij> J_ij delta(s_i, s_j) for cfg (..., L, L) of integers."""
    c = np.asarray(cfg)
    e = -(Jr[..., :, :-1] * (c[..., :, :-1] == c[..., :, 1:])).sum(axis=(-1, -2))
    e = e - (Jd[..., :-1, :] * (c[..., :-1, :] == c[..., 1:, :])).sum(axis=(-1, -2))
    return e


def brute_force(Jr, Jd, beta, q):
    """all q^(L*L) configurations (raster order, site 0 slowest), energies, log Z, Boltzmann probabilities."""
    L = Jr.shape[0]
    cfgs = np.array(list(itertools.product(range(q), repeat=L * L)), dtype=np.int8).reshape(-1, L, L)
    E = energy(cfgs, Jr, Jd).astype(float)
    w = -beta * E
    m = w.max()
    logZ = m + np.log(np.exp(w - m).sum())
    return cfgs, E, logZ, np.exp(w - logZ)


def sample_row(mps, cfg_up, J_up, beta, u_row, q, forced_row=None):
    """PAPER.md:220-254 with q outcomes per site.  Returns (row_cfgs (bs,L), row log-probs (bs,), probs (bs,L,q))."""
    L = len(mps)
    bs = cfg_up.shape[0]
    row_cfgs = np.zeros((bs, L), dtype=np.int8)
    logp = np.zeros(bs)
    probs_out = np.zeros((bs, L, q))
    right = {L - 1: np.ones((bs, 1))}
    for col in range(L - 2, -1, -1):                       # right environments given the upper row
        Bm = potts_bmat(beta, J_up[col + 1], q)
        tmp = np.einsum("ijk,lj->ilk", mps[col + 1], Bm)[:, cfg_up[:, col + 1].astype(np.int64), :]
        right[col] = np.einsum("ibj,bj->bi", tmp, right[col + 1])
        right[col] /= np.linalg.norm(right[col], axis=1, keepdims=True)
    left = np.ones((bs, 1))
    for col in range(L):                                   # left sampling sweep
        rho = np.abs(np.einsum("bi,ijk,bk->bj", left, mps[col], right[col]))          # (bs, q)
        w = rho * potts_bmat(beta, J_up[col], q)[cfg_up[:, col].astype(np.int64), :]    # weight of the up bond
        p = w / w.sum(axis=1, keepdims=True)
        if forced_row is None:
            a = (np.cumsum(p, axis=1)[:, :-1] <= u_row[:, col][:, None]).sum(axis=1)
        else:
            a = forced_row[:, col].astype(np.int64)
        row_cfgs[:, col] = a
        probs_out[:, col, :] = p
        logp += np.log(p[np.arange(bs), a])
        left = np.einsum("bi,ibj->bj", left, mps[col][:, a, :])
        left /= np.linalg.norm(left, axis=1, keepdims=True)
    return row_cfgs, logp, probs_out


def sample(cache, Jd, beta, u, q, forced=None):
    """cfgs (bs,L,L), log q (bs,), probs (bs,L,L,q)."""
    L = len(cache)
    bs = u.shape[0]
    cfgs = np.zeros((bs, L, L), dtype=np.int8)
    logq = np.zeros(bs)
    probs = np.zeros((bs, L, L, q))
    for row in range(L):
        if row == 0:
            cfg_up = np.zeros((bs, L), dtype=np.int8); J_up = np.zeros(L)
        else:
            cfg_up = cfgs[:, row - 1, :]; J_up = Jd[row - 1, :]
        rc, lp, pr = sample_row(cache[row], cfg_up, J_up, beta, u[:, row, :], q,
                                None if forced is None else forced[:, row, :])
        cfgs[:, row, :] = rc
        logq += lp
        probs[:, row] = pr
    return cfgs, logq, probs
