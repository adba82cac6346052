"""Oracle Part S: row-by-row ancestral sampling (test infrastructure, see oracle/__init__.py).

Follows `SamplerIsing.sample` / `_sample_row` step by step for ONE
disorder realisation, batched over `bs` samples exactly as the listing is.  numpy, FP64
(the listing is torch.float; reading G14 of DESIGN.md).

Differences from the listing, all readings listed in DESIGN.md:
  * the random draw: u < p with u passed in (Philox uniforms, oracle/philox.py) replaces
    `Bernoulli(probs).sample()`; same semantics (spin up iff u < p);
  * log-prob in the stable form  log sigma(+-x)  without torch's eps clamp (G13);
  * row 0 has no upper row: J_up = 0 so B = 1 and up_field = 0 (G9; the listing reads the
    wrapped-around all-False row with the zero boundary coupling, same effect);
  * optional teacher forcing (`forced`): use the given spins instead of u < p, still
    returning log q and the conditional probabilities.
"""
import numpy as np

from .bmps import set_ising_bmat


def sample_row(mps, cfg_up, J_up, beta, u_row, forced_row=None):
    """PAPER.md:220-254. mps: list of L tensors (D_l,2,D_r); cfg_up: (bs,L) in {0,1};
    J_up: (L,) up couplings of this row; u_row: (bs,L) uniforms.
    Returns row_cfgs (bs,L) int8, row_log_probs (bs,), probs (bs,L)."""
    L = len(mps)
    bs = cfg_up.shape[0]
    row_cfgs = np.zeros((bs, L), dtype=np.int8)
    row_log_probs = np.zeros((bs, L))
    probs_out = np.zeros((bs, L))
    # right environments given the upper row and the Boltzmann weights
    right_envs = {L - 1: np.ones((bs, 1))}
    for col in range(L - 2, -1, -1):
        B_mat = set_ising_bmat(beta, J_up[col + 1])
        tmp = np.einsum("ijk,lj->ilk", mps[col + 1], B_mat)
        tmp = tmp[:, cfg_up[:, col + 1].astype(np.int64), :]              # (D_l, bs, D_r)
        right_envs[col] = np.einsum("ibj,bj->bi", tmp, right_envs[col + 1])
        right_envs[col] /= np.linalg.norm(right_envs[col], axis=1, keepdims=True)
    # sampling from left to right
    left_env = np.ones((bs, 1))
    for col in range(L):
        rho = np.abs(np.einsum("bi,ijk,bk->bj", left_env, mps[col], right_envs[col]))   # (bs,2)
        up_field = 2.0 * beta * float(J_up[col]) * (2.0 * cfg_up[:, col] - 1.0)
        x = np.log(rho[:, 1] / rho[:, 0]) + up_field
        probs = 1.0 / (1.0 + np.exp(-x))                                   # sigmoid, Eq. 5
        if forced_row is None:
            a = (u_row[:, col] < probs).astype(np.int8)
        else:
            a = forced_row[:, col].astype(np.int8)
        row_cfgs[:, col] = a
        probs_out[:, col] = probs
        row_log_probs[:, col] = np.where(a == 1, -np.log1p(np.exp(-x)), -np.log1p(np.exp(x)))
        left_env = np.einsum("bi,ibj->bj", left_env, mps[col][:, a.astype(np.int64), :])
        left_env /= np.linalg.norm(left_env, axis=1, keepdims=True)
    return row_cfgs, row_log_probs.sum(axis=1), probs_out


def sample(cache, Jd, beta, u, forced=None):
    """PAPER.md:202-217. cache[r] = MPS of rows r..L-1; Jd: (L,L); u: (bs,L,L) uniforms.
    Returns cfgs (bs,L,L) int8, log_probs (bs,), probs (bs,L,L) = q(s_i=+1 | s_<i)."""
    L = len(cache)
    bs = u.shape[0]
    cfgs = np.zeros((bs, L, L), dtype=np.int8)
    log_probs = np.zeros(bs)
    probs = np.zeros((bs, L, L))
    for row in range(L):
        if row == 0:
            cfg_up = np.zeros((bs, L), dtype=np.int8); J_up = np.zeros(L)
        else:
            cfg_up = cfgs[:, row - 1, :]; J_up = Jd[row - 1, :]
        row_cfgs, row_log_probs, row_probs = sample_row(
            cache[row], cfg_up, J_up, beta, u[:, row, :],
            None if forced is None else forced[:, row, :])
        cfgs[:, row, :] = row_cfgs
        log_probs += row_log_probs
        probs[:, row, :] = row_probs
    return cfgs, log_probs, probs
