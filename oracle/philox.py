"""Oracle Part R: counter-based uniforms (test infrastructure, see oracle/__init__.py).

The paper draws spins with `Bernoulli(probs).sample()` from torch's global RNG
(PAPER.md:247-248), which fixes nothing reproducible.  BASELINE.json north_star asks
for "Philox counter-based uniforms indexed by (disorder, sample, site)".  Reading R
(DESIGN.md): Philox4x32-10 (Salmon et al., SC'11), restated here from the published
algorithm: 10 rounds of
    (c0,c1,c2,c3) <- (hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0))
with M0=0xD2511F53, M1=0xCD9E8D57, and the key bumped by (0x9E3779B9, 0xBB67AE85)
between rounds.

Indexing (reading R):
    key     = (seed & 0xffffffff, seed >> 32)
    counter = (site = r*L + c, sample index, disorder index, tag)
    tag 0 = spin draws, tag 1 = Metropolis draws (site word 0, sample word = step index)
    u = ((x0 << 21) | (x1 >> 11)) * 2**-53  in [0,1)  from output words x0, x1
A spin is +1 iff u < p (torch.bernoulli semantics of PAPER.md:247-248).
"""
import numpy as np

M0 = np.uint64(0xD2511F53)
M1 = np.uint64(0xCD9E8D57)
W0 = 0x9E3779B9
W1 = 0xBB67AE85
MASK32 = np.uint64(0xFFFFFFFF)
TAG_SPIN = 0
TAG_METROPOLIS = 1


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds on broadcastable uint32 arrays -> 4 uint32 arrays."""
    c0, c1, c2, c3 = (np.asarray(x, dtype=np.uint64) & MASK32 for x in (c0, c1, c2, c3))
    c0, c1, c2, c3 = np.broadcast_arrays(c0, c1, c2, c3)
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = M0 * c0                      # 64-bit product of two 32-bit values
        p1 = M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & MASK32
        hi1, lo1 = p1 >> np.uint64(32), p1 & MASK32
        c0, c1, c2, c3 = (hi1 ^ c1 ^ np.uint64(k0), lo1, hi0 ^ c3 ^ np.uint64(k1), lo0)
        k0 = (k0 + W0) & 0xFFFFFFFF
        k1 = (k1 + W1) & 0xFFFFFFFF
    return tuple(x.astype(np.uint32) for x in (c0, c1, c2, c3))


def uniform53(x0, x1):
    """53-bit uniform in [0,1): high 32 bits from x0, low 21 bits from the top of x1."""
    m = (np.asarray(x0, dtype=np.uint64) << np.uint64(21)) | (np.asarray(x1, dtype=np.uint64) >> np.uint64(11))
    return m.astype(np.float64) * 2.0 ** -53


def spin_uniforms(seed, disorder, samples, site):
    """u[(samples...)] for spin draws at one (disorder, site); `samples` = global sample indices."""
    x0, x1, _, _ = philox4x32_10(site, samples, disorder, TAG_SPIN, seed & 0xFFFFFFFF, seed >> 32)
    return uniform53(x0, x1)


def metropolis_uniforms(seed, disorder, steps):
    """u[(steps...)] for the Metropolis accept draws of one disorder's chain."""
    x0, x1, _, _ = philox4x32_10(0, steps, disorder, TAG_METROPOLIS, seed & 0xFFFFFFFF, seed >> 32)
    return uniform53(x0, x1)
