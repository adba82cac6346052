"""GPU parity, third part: the chi=32 kernels (256-thread CTAs, M kept in the L2 scratch) against the
oracle at a size it finishes in seconds, and config C3 (128x128, chi=32, 256 x 256) at full size in the
launch configuration bench.py times, checked on sampled outputs the oracle can compute one by one
(energies, Metropolis scan) and on properties that hold at any size (teacher-forced log q reproduces
the sampled log q bit for bit; chunked calls agree; fault counters stay at zero)."""
import numpy as np
import pytest

from oracle import bmps, exact, metropolis, philox, sampler
from tnmc_workloads import CONFIGS, make_couplings

from bitpack import unpack
import noise_floor as nf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tn():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2509_19006_b200 import tnmc
    return tnmc


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


@pytest.mark.parametrize("L,chi,beta,n_dis,n_s,seed", [(40, 32, 1.0, 2, 24, 41), (24, 32, 0.7, 2, 130, 42), (33, 20, 1.5, 1, 16, 43)])
def test_chi32_parity(tn, L, chi, beta, n_dis, n_s, seed):
    """bond dimensions above 16 run the P = 32 instantiation: log Z, conditionals, spins, log q, energies."""
    dev = torch.device("cuda:0")
    Jr, Jd = make_couplings(L, n_dis, seed)
    ctx = tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s)
    logZ = ctx.tnmc_build_envs().cpu().numpy()
    probs = torch.zeros((n_dis, n_s, L, L), dtype=torch.float64, device=dev)
    bits, logq = ctx.tnmc_sample(n_s, seed, probs=probs)
    E = ctx.tnmc_energy(bits).cpu().numpy()
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["rho_zero"] == 0 and flags["logz_nonpos"] == 0
    cfg = unpack(_u32(bits), L)
    n_chk = min(n_s, 24)
    for d in range(n_dis):
        cache, ls = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        cache_p, ls_p = nf.perturbed_cache(Jr[d], Jd[d], beta, chi)
        lz, sign = bmps.log_z(cache[0], ls[0])
        assert sign == 1.0
        assert abs(logZ[d] - lz) <= nf.tol(1e-10 * abs(lz), nf.logz_floor(cache, ls, cache_p, ls_p))
        u = np.empty((n_chk, L, L))
        for r in range(L):
            for c in range(L):
                u[:, r, c] = philox.spin_uniforms(seed, d, np.arange(n_chk), r * L + c)
        o_cfg, o_logq, o_probs = sampler.sample(cache, Jd[d], beta, u)
        fl_p, fl_q = nf.probs_floor(cache_p, Jd[d], beta, o_cfg, o_probs, o_logq)
        tol_p = nf.tol(1e-9, fl_p)
        same = (cfg[d, :n_chk] == o_cfg).all(axis=(1, 2))
        near = (np.abs(u - o_probs) < tol_p).any(axis=(1, 2))
        assert (same | near).all()
        ok = same & ~near
        assert ok.sum() >= n_chk - 2
        assert np.abs(probs[d, :n_chk].cpu().numpy()[ok] - o_probs[ok]).max() < tol_p
        assert np.abs(logq[d, :n_chk].cpu().numpy()[ok] - o_logq[ok]).max() < nf.tol(1e-9 * np.abs(o_logq).max(), fl_q)
        assert (E[d, :n_chk][ok] == exact.energy(o_cfg[ok], Jr[d], Jd[d])).all()


def test_config_c3_full_size(tn):
    """Config C3 exactly as bench.py launches it (256 disorders x 256 samples, full stack, one workspace)."""
    c = CONFIGS["C3"]
    L, chi, beta, n_dis, n_s = c["L"], c["chi"], c["betas"][0], c["n_dis"], c["n_samples"]
    dev = torch.device("cuda:0")
    free, _ = torch.cuda.mem_get_info()
    need = tn.tnmc_workspace_bytes(L, chi, n_dis, n_s)
    if free < need + (8 << 30):
        pytest.skip("not enough free HBM for the full C3 stack")
    Jr, Jd = make_couplings(L, n_dis, c["inst_seed"])
    ctx = tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s)
    logZ = ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, c["seed"])
    E = ctx.tnmc_energy(bits)
    acc, n_acc, state, _ = ctx.tnmc_metropolis(E, logq, c["seed"])
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["rho_zero"] == 0 and flags["logz_nonpos"] == 0
    assert torch.isfinite(logZ).all() and torch.isfinite(logq).all()
    # log Z per site of the +-J model at beta = 1 lies between the ground-state bound and the free-spin bound
    per_site = (logZ / (L * L)).cpu().numpy()
    assert (per_site > np.log(2.0)).all() and (per_site < np.log(2.0) + 2.0 * np.log(np.cosh(beta))).all()
    # sampled outputs the oracle computes one by one: energies (bit-exact) and the Metropolis scan
    E_h, q_h, acc_h = E.cpu().numpy(), logq.cpu().numpy(), acc.cpu().numpy()
    for d in (0, 101, 255):
        cfg = unpack(_u32(bits[d, :32]), L)
        assert (E_h[d, :32] == exact.energy(cfg, Jr[d], Jd[d])).all()
        um = philox.metropolis_uniforms(c["seed"], d, np.arange(n_s))
        o_acc, o_n, cE, cq, ci, _ = metropolis.metropolis_scan(E_h[d], q_h[d], beta, um)
        assert (acc_h[d] == o_acc).all() and int(n_acc[d]) == o_n
        assert int(state[1][d]) == cE and int(state[2][d]) == ci
    # property: teacher-forcing the sampler on its own configurations reproduces log q bit for bit,
    # and a chunk of disorders / samples reproduces the same spins (Philox indexing)
    sl = slice(100, 104)
    b2, q2 = ctx.tnmc_sample(n_s, c["seed"], dis_begin=100, dis_count=4, forced_cfg_bits=bits[sl].contiguous())
    assert torch.equal(b2, bits[sl]) and torch.equal(q2, logq[sl])
    b3, q3 = ctx.tnmc_sample(64, c["seed"], sample_offset=128, dis_begin=200, dis_count=3)
    assert torch.equal(b3, bits[200:203, 128:192]) and torch.equal(q3, logq[200:203, 128:192])
    # truncated proposal: acceptance is high but log q is not the Boltzmann weight exactly
    p_acc = float(n_acc.sum()) / (n_dis * (n_s - 1))
    assert 0.5 < p_acc <= 1.0
