"""Pins 8 and 10: Metropolis scan and the Philox generator of the oracle."""
import os
import shutil
import subprocess

import numpy as np
import pytest

from oracle import bmps, exact, metropolis, philox, sampler
from tnmc_workloads import make_couplings

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers():
    for line in open(os.path.join(GOLD, "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        out = philox.philox4x32_10(w[0], w[1], w[2], w[3], w[4], w[5])
        assert [int(x) for x in out] == w[6:]


CURAND_SRC = r"""
#include <cstdio>
#include <cstdint>
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
int main() {
  // counters on a lattice of (site, sample, disorder, tag) words, two keys
  for (unsigned key = 0; key < 2; ++key)
    for (unsigned tag = 0; tag < 2; ++tag)
      for (unsigned d = 0; d < 5; ++d)
        for (unsigned n = 0; n < 100; ++n)
          for (unsigned site = 0; site < 100; ++site) {
            uint4 c; c.x = site * 2654435761u; c.y = n * 40503u + 7u; c.z = d * 1000003u; c.w = tag;
            uint2 k; k.x = key ? 0xdeadbeefu : 2002u; k.y = key ? 0x12345678u : 0u;
            uint4 r = curand_Philox4x32_10(c, k);
            printf("%u %u %u %u\n", r.x, r.y, r.z, r.w);
          }
}
"""


@pytest.mark.skipif(shutil.which("g++") is None or not os.path.exists("/usr/local/cuda/include/curand_philox4x32_x.h"),
                    reason="needs g++ and the CUDA toolkit headers")
def test_philox_against_curand_header(tmp_path):
    """Pin 10: 10^5 counters against cuRAND's own Philox4x32-10 (header compiled for the host)."""
    src = tmp_path / "ph.cpp"
    src.write_text(CURAND_SRC)
    exe = tmp_path / "ph"
    subprocess.check_call(["g++", "-O2", "-I/usr/local/cuda/include", str(src), "-o", str(exe)])
    ref = np.array(subprocess.check_output([str(exe)]).split(), dtype=np.uint64).reshape(-1, 4)
    key, tag, d, n, site = np.meshgrid(np.arange(2), np.arange(2), np.arange(5), np.arange(100), np.arange(100), indexing="ij")
    c0 = (site.astype(np.uint64) * 2654435761) & 0xFFFFFFFF
    c1 = (n.astype(np.uint64) * 40503 + 7) & 0xFFFFFFFF
    c2 = (d.astype(np.uint64) * 1000003) & 0xFFFFFFFF
    got = np.zeros(ref.shape, dtype=np.uint64)
    for kk, (k0, k1) in enumerate([(2002, 0), (0xdeadbeef, 0x12345678)]):
        sel = key == kk
        out = philox.philox4x32_10(c0[sel], c1[sel], c2[sel], tag[sel], k0, k1)
        got[sel.reshape(-1)] = np.stack(out, axis=1)
    assert (got == ref).all()


def test_uniform_construction_and_moments():
    assert philox.uniform53(0, 0) == 0.0
    assert philox.uniform53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    assert philox.uniform53(0x80000000, 0) == 0.5
    assert philox.uniform53(0, 1 << 11) == 2.0 ** -53
    u = philox.spin_uniforms(2002, 3, np.arange(200000), 17)
    assert (u >= 0).all() and (u < 1).all()
    assert abs(u.mean() - 0.5) < 4 * np.sqrt(1 / 12 / u.size)
    assert abs(u.var() - 1 / 12) < 0.002
    # indexing: distinct (disorder, sample, site, tag) give distinct streams
    a = philox.spin_uniforms(2002, 3, np.arange(10), 17)
    assert not np.allclose(a, philox.spin_uniforms(2002, 4, np.arange(10), 17))
    assert not np.allclose(a, philox.spin_uniforms(2002, 3, np.arange(10), 18))
    assert not np.allclose(a, philox.spin_uniforms(2003, 3, np.arange(10), 17))
    assert not np.allclose(philox.spin_uniforms(2002, 3, np.arange(10), 0), philox.metropolis_uniforms(2002, 3, np.arange(10)))
    assert np.array_equal(a[3:6], philox.spin_uniforms(2002, 3, np.arange(3, 6), 17))


def test_metropolis_hand_worked():
    """Pin 8: the hand-worked chain of tests/golden/metropolis_hand.txt."""
    g = {}
    for line in open(os.path.join(GOLD, "metropolis_hand.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        g[k] = v
    beta = float(g["beta"][0])
    E = np.array(g["E"], dtype=np.int64)
    logq = np.array(g["logq"], dtype=np.float64)
    u = np.array(g["u"], dtype=np.float64)
    acc, n_acc, cE, clq, cidx, sr = metropolis.metropolis_scan(E, logq, beta, u)
    assert list(acc) == [int(x) for x in g["accepted"]]
    assert n_acc == int(g["n_accepted"][0])
    assert (cE, clq, cidx) == (int(g["final"][0]), float(g["final"][1]), int(g["final"][2]))
    assert sr == pytest.approx(2 * np.exp(-3.0) + 2.0, rel=1e-15)
    # continuing a chain in two calls gives the same result as one call
    a1 = metropolis.metropolis_scan(E[:2], logq[:2], beta, u[:2])
    a2 = metropolis.metropolis_scan(E[2:], logq[2:], beta, u[2:], a1[2], a1[3], a1[4], idx_offset=2)
    assert list(a1[0]) + list(a2[0]) == list(acc) and a2[4] == cidx and a1[1] + a2[1] == n_acc


def test_metropolis_exact_chi_accepts_everything():
    """Pin 8 / PAPER.md:284: P_acc = 1 iff the proposal is the Boltzmann distribution."""
    L, beta = 6, 1.0
    Jr, Jd = make_couplings(L, 1, 41); Jr, Jd = Jr[0], Jd[0]
    cache, _ = bmps.build_cache(Jr, Jd, beta, 8)
    n = 64
    u = np.stack([[philox.spin_uniforms(5, 0, np.arange(n), r * L + c) for c in range(L)] for r in range(L)])
    cfgs, logq, _ = sampler.sample(cache, Jd, beta, np.transpose(u, (2, 0, 1)))
    E = exact.energy(cfgs, Jr, Jd)
    um = philox.metropolis_uniforms(5, 0, np.arange(n))
    # |logA| is rounding noise (~1e-12): nudge u away from 1 so that log u < logA is decided by the physics
    acc, n_acc, *_ , sr = metropolis.metropolis_scan(E, logq, beta, np.minimum(um, 1 - 1e-9))
    assert n_acc == n - 1 and acc.all()
    assert sr == pytest.approx(n - 1, abs=1e-8)


def test_metropolis_truncated_chain_converges_to_boltzmann():
    """Pin 8 (statistical): 3x3, chi = 2 truncated proposal, long chain histogram -> Boltzmann."""
    L, beta = 3, 1.0
    Jr, Jd = make_couplings(L, 1, 43); Jr, Jd = Jr[0], Jd[0]
    Jr = np.abs(Jr); Jd = np.abs(Jd)          # ferromagnet: chi = 1 truncation is visibly inexact
    cache, _ = bmps.build_cache(Jr, Jd, beta, 1)
    n = 60000
    u = np.zeros((n, L, L))
    for r in range(L):
        for c in range(L):
            u[:, r, c] = philox.spin_uniforms(77, 0, np.arange(n), r * L + c)
    cfgs, logq, _ = sampler.sample(cache, Jd, beta, u)
    E = exact.energy(cfgs, Jr, Jd)
    um = philox.metropolis_uniforms(77, 0, np.arange(n))
    acc, n_acc, *_ = metropolis.metropolis_scan(E, logq, beta, um)
    assert 0.05 < n_acc / (n - 1) < 0.999          # truncation makes the proposal inexact
    # chain state at every step = last accepted proposal
    idx = np.maximum.accumulate(np.where(acc == 1, np.arange(n), 0))
    code = (cfgs.reshape(n, -1) * (1 << np.arange(L * L - 1, -1, -1))).sum(axis=1)
    _, _, _, P = exact.brute_force(Jr, Jd, beta)
    burn = 1000
    chain_hist = np.bincount(code[idx][burn:], minlength=512) / (n - burn)
    prop_hist = np.bincount(code[burn:], minlength=512) / (n - burn)
    # total-variation distance: the corrected chain is close to Boltzmann, the raw proposal is not
    tv_chain = 0.5 * np.abs(chain_hist - P).sum()
    tv_prop = 0.5 * np.abs(prop_hist - P).sum()
    assert tv_chain < 0.03
    assert tv_prop > 2 * tv_chain
