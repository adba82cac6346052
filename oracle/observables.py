"""Oracle: thermal averages along the Metropolis chain (test infrastructure, see oracle/__init__.py).

The paper's samples exist to estimate observables of the Boltzmann distribution (PAPER.md:23, :39:
"unbiased samples ... physical observables"); it shows no code for this step.  Reading G19
(DESIGN.md): the estimator is the plain MCMC average over chain STEPS -- at step n the chain sits on
the last accepted proposal (Eq. 10; readings G15/G16), and every step counts once,
rejected steps re-counting the state they stayed on.  Observables per configuration:
  E   Eq. 1, integer
  M   = sum_i s_i (magnetisation, integer in [-N, N])
accumulated as the five sums  sum E, sum E^2, sum M, sum |M|, sum M^2  over the steps of a chunk.

Replica overlap (the spin-glass order parameter; the +-J Edwards-Anderson model of PAPER.md:282-286 has
<M> = 0 by symmetry, so the overlap between two independent replicas of the SAME disorder is the observable
that carries the physics):  q = sum_i s_i^a s_i^b  (integer in [-N, N]; q/N is the usual normalisation).
Two independent Metropolis chains a, b (different Philox sample ranges or seeds) are walked step by step;
at step n each sits on its last accepted proposal, q_n is the overlap of the two current states, and the
sums  sum q, sum |q|, sum q^2  are accumulated like the five above (same reading G19).
"""
import numpy as np


def magnetisation(cfg):
    """M = sum_i s_i for cfg (..., L, L) in {0,1}."""
    c = np.asarray(cfg, dtype=np.int64)
    return (2 * c - 1).sum(axis=(-1, -2))


def chain_sums(E, M, accepted, cur_E=0, cur_M=0):
    """E, M: (n,) ints of the proposals; accepted: (n,) flags from the Metropolis scan (flag 1 on the
    proposal that initialises an empty chain).  cur_E / cur_M: state entering the chunk (used until the
    first flag 1).  Returns (sums[5] as Python ints, cur_E, cur_M)."""
    s = [0, 0, 0, 0, 0]
    for i in range(len(E)):
        if accepted[i]:
            cur_E, cur_M = int(E[i]), int(M[i])
        s[0] += cur_E
        s[1] += cur_E * cur_E
        s[2] += cur_M
        s[3] += abs(cur_M)
        s[4] += cur_M * cur_M
    return s, cur_E, cur_M


def chain_sums_real(E, M, accepted, cur_E=0.0, cur_M=0):
    """As chain_sums for real-valued energies (real couplings): sums of E and E^2 as floats in proposal order."""
    s = [0.0, 0.0, 0, 0, 0]
    for i in range(len(E)):
        if accepted[i]:
            cur_E, cur_M = float(E[i]), int(M[i])
        s[0] += cur_E
        s[1] += cur_E * cur_E
        s[2] += cur_M
        s[3] += abs(cur_M)
        s[4] += cur_M * cur_M
    return s, cur_E, cur_M


def overlap(cfg_a, cfg_b):
    """q = sum_i s_i^a s_i^b for cfg (..., L, L) in {0,1}: N - 2 * (number of sites where the two differ)."""
    a = 2 * np.asarray(cfg_a, dtype=np.int64) - 1
    b = 2 * np.asarray(cfg_b, dtype=np.int64) - 1
    return (a * b).sum(axis=(-1, -2))


def replica_overlap(cfg_a, acc_a, cfg_b, acc_b, cur_a=None, cur_b=None):
    """cfg_x: (n, L, L) proposals of chain x, acc_x: (n,) Metropolis flags of chain x (flag 1 on the proposal that
    initialises an empty chain); cur_x: (L, L) state of chain x entering the chunk (used until its first flag 1).
    Returns (q_steps (n,) int64, sums [sum q, sum |q|, sum q^2] as Python ints, cur_a, cur_b)."""
    n = len(acc_a)
    q = np.zeros(n, dtype=np.int64)
    s = [0, 0, 0]
    for i in range(n):
        if acc_a[i]:
            cur_a = np.asarray(cfg_a[i])
        if acc_b[i]:
            cur_b = np.asarray(cfg_b[i])
        qi = int(overlap(cur_a, cur_b))
        q[i] = qi
        s[0] += qi
        s[1] += abs(qi)
        s[2] += qi * qi
    return q, s, cur_a, cur_b
