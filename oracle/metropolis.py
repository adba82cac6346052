"""Oracle Part S4: independence Metropolis-Hastings scan (test infrastructure).

Eq. 10:  P_acc(s -> s') = min[1, q(s) e^{-beta E(s')} / (q(s') e^{-beta E(s)})].
The paper shows no code for this step.  Readings G15/G16: one chain per disorder,
proposals taken in sample-index order; a chain with cur_idx < 0 is empty and its first
proposal initialises it (flag 1, not counted as an acceptance); accept iff
log u < logA with  logA = -beta (E' - E) + log q(s) - log q(s'),  u in [0,1), log 0 = -inf.
"""
import numpy as np


def metropolis_scan(E, logq, beta, u, cur_E=0, cur_logq=0.0, cur_idx=-1, idx_offset=0):
    """E: (n,) ints, logq: (n,) floats, u: (n,) uniforms (u[0] unused when the chain is empty).
    Returns (accepted (n,) uint8, n_accepted, cur_E, cur_logq, cur_idx, sum_min1_ratio)."""
    n = len(E)
    accepted = np.zeros(n, dtype=np.uint8)
    n_acc = 0
    sum_ratio = 0.0
    for i in range(n):
        if cur_idx < 0:
            cur_E, cur_logq, cur_idx = int(E[i]), float(logq[i]), idx_offset + i
            accepted[i] = 1
            continue
        logA = -beta * float(int(E[i]) - cur_E) + cur_logq - float(logq[i])
        sum_ratio += min(1.0, np.exp(min(logA, 0.0)))
        logu = np.log(u[i]) if u[i] > 0.0 else -np.inf
        if logu < logA:
            cur_E, cur_logq, cur_idx = int(E[i]), float(logq[i]), idx_offset + i
            accepted[i] = 1
            n_acc += 1
    return accepted, n_acc, cur_E, cur_logq, cur_idx, sum_ratio


def metropolis_scan_real(E, logq, beta, u, cur_E=0.0, cur_logq=0.0, cur_idx=-1, idx_offset=0):
    """The same scan for real-valued energies (real couplings): Eq. 10 unchanged."""
    n = len(E)
    accepted = np.zeros(n, dtype=np.uint8)
    n_acc = 0
    sum_ratio = 0.0
    for i in range(n):
        if cur_idx < 0:
            cur_E, cur_logq, cur_idx = float(E[i]), float(logq[i]), idx_offset + i
            accepted[i] = 1
            continue
        logA = -beta * (float(E[i]) - cur_E) + cur_logq - float(logq[i])
        sum_ratio += min(1.0, np.exp(min(logA, 0.0)))
        logu = np.log(u[i]) if u[i] > 0.0 else -np.inf
        if logu < logA:
            cur_E, cur_logq, cur_idx = float(E[i]), float(logq[i]), idx_offset + i
            accepted[i] = 1
            n_acc += 1
    return accepted, n_acc, cur_E, cur_logq, cur_idx, sum_ratio
