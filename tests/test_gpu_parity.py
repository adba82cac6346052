"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star's: energies and spins
drawn with the same uniforms bit-exact (except draws within 1e-9 of a threshold, counted);
log Z relative 1e-10; conditional probabilities absolute 1e-9."""
import numpy as np
import pytest

from oracle import bmps, exact, metropolis, philox, sampler
from tnmc_workloads import make_couplings

from bitpack import pack, unpack
import noise_floor as nf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tn():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2509_19006_b200 import tnmc
    return tnmc


def _ctx(tn, L, chi, beta, Jr, Jd, n_samples_max, **kw):
    dev = torch.device("cuda:0")
    return tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_samples_max, **kw)


def _oracle_uniforms(seed, d, n_samples, L, sample_offset=0):
    samples = np.arange(sample_offset, sample_offset + n_samples)
    u = np.empty((n_samples, L, L))
    for r in range(L):
        for c in range(L):
            u[:, r, c] = philox.spin_uniforms(seed, d, samples, r * L + c)
    return u


def _to_np_u32(t):
    return t.cpu().numpy().view(np.uint32)


# ------------------------------------------------------------------------------------------ energy
@pytest.mark.parametrize("L,n_dis,n_s", [(2, 3, 5), (8, 4, 64), (31, 3, 17), (33, 2, 9), (64, 2, 8), (70, 2, 11), (128, 2, 6)])
def test_energy_bit_exact(tn, L, n_dis, n_s):
    rng = np.random.default_rng(L * 1000 + n_s)
    Jr, Jd = make_couplings(L, n_dis, 77 + L)
    if L == 31:   # diluted bonds (J = 0 allowed by the ABI)
        Jr[rng.random(Jr.shape) < 0.2] = 0
        Jd[rng.random(Jd.shape) < 0.2] = 0
    cfg = rng.integers(0, 2, (n_dis, n_s, L, L)).astype(np.int8)
    cfg[0, 0] = 1
    cfg[0, 1 % n_s] = 0
    ctx = _ctx(tn, L, 4, 1.0, Jr, Jd, n_s)
    bits = torch.from_numpy(pack(cfg).view(np.int32)).cuda()
    E = ctx.tnmc_energy(bits).cpu().numpy()
    for d in range(n_dis):
        assert (E[d] == exact.energy(cfg[d], Jr[d], Jd[d])).all()
    # sub-range of disorders
    if n_dis > 1:
        E1 = ctx.tnmc_energy(bits[1:].contiguous(), dis_begin=1).cpu().numpy()
        assert (E1 == E[1:]).all()


# ------------------------------------------------------------------------------------------ build
CASES_BUILD = [
    # L, chi, beta, n_dis, seed
    (2, 2, 1.0, 2, 1),
    (3, 2, 0.7, 2, 2),
    (4, 4, 1.0, 3, 3),       # exact chi
    (4, 2, 1.0, 3, 4),       # truncated
    (6, 3, 0.5, 2, 5),       # chi not a power of two
    (8, 16, 1.0, 4, 1001),   # config C1 (exact chi)
    (8, 4, 2.0, 2, 6),
    (12, 8, 1.0, 2, 7),
    (13, 5, 1.3, 2, 8),      # odd L, odd chi
]


@pytest.mark.parametrize("L,chi,beta,n_dis,seed", CASES_BUILD)
def test_build_logz_and_states(tn, L, chi, beta, n_dis, seed):
    Jr, Jd = make_couplings(L, n_dis, seed)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, 8)
    logZ = ctx.tnmc_build_envs().cpu().numpy()
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["logz_nonpos"] == 0
    for d in range(n_dis):
        cache, ls = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        cache_p, ls_p = nf.perturbed_cache(Jr[d], Jd[d], beta, chi)
        floor = nf.state_floor(cache, cache_p)
        lz, sign = bmps.log_z(cache[0], ls[0])
        assert sign == 1.0
        assert abs(logZ[d] - lz) <= nf.tol(1e-10 * abs(lz), nf.logz_floor(cache, ls, cache_p, ls_p))
        for r in range(L):
            row, lsr = ctx.tnmc_get_env_row(d, r)
            row = row.numpy()
            # gauge-invariant comparison: expand both to the 2^L vector (the stored state has a definite sign)
            mps = []
            for c in range(L):
                dl, dr = cache[r][c].shape[0], cache[r][c].shape[2]
                assert np.abs(row[c][dl:, :, :]).max(initial=0.0) == 0.0 and np.abs(row[c][:, :, dr:]).max(initial=0.0) == 0.0
                mps.append(row[c][:dl, :, :dr])
            v_gpu = bmps.mps_to_vector(mps)
            v_cpu = bmps.mps_to_vector(cache[r])
            scale = np.abs(v_cpu).max()
            tol = nf.tol(1e-10, floor[r], cap=(L, chi, beta) != (13, 5, 1.3))   # the one deliberately ill-conditioned case
            assert np.abs(v_gpu - v_cpu).max() <= tol * scale
            assert abs(lsr - ls[r]) <= tol * max(1.0, abs(ls[r]))


# ------------------------------------------------------------------------------------------ sampling
CASES_SAMPLE = [
    # L, chi, beta, n_dis, n_samples, seed
    (2, 2, 1.0, 2, 5, 11),
    (4, 4, 1.0, 2, 33, 12),      # exact
    (4, 2, 1.0, 2, 130, 13),     # truncated, more than one chain tile, ragged
    (6, 3, 0.5, 2, 17, 14),
    (8, 16, 1.0, 4, 64, 2001),   # config C1
    (12, 8, 2.0, 2, 40, 15),
    (33, 8, 1.0, 1, 20, 16),     # two bit words per row
]


@pytest.mark.parametrize("L,chi,beta,n_dis,n_s,seed", CASES_SAMPLE)
def test_sample_parity(tn, L, chi, beta, n_dis, n_s, seed):
    Jr, Jd = make_couplings(L, n_dis, seed + 100)
    first = 5
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s, first_disorder=first)
    ctx.tnmc_build_envs()
    probs = torch.zeros((n_dis, n_s, L, L), dtype=torch.float64, device="cuda")
    off = 3
    bits, logq = ctx.tnmc_sample(n_s, seed, sample_offset=off, probs=probs)
    flags = ctx.tnmc_get_flags()
    cfg = unpack(_to_np_u32(bits), L)
    logq = logq.cpu().numpy()
    probs = probs.cpu().numpy()
    E = ctx.tnmc_energy(bits).cpu().numpy()
    n_near = 0
    for d in range(n_dis):
        cache, _ = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        u = _oracle_uniforms(seed, first + d, n_s, L, off)
        o_cfg, o_logq, o_probs = sampler.sample(cache, Jd[d], beta, u)
        cache_p, _ = nf.perturbed_cache(Jr[d], Jd[d], beta, chi)
        fl_p, fl_q = nf.probs_floor(cache_p, Jd[d], beta, o_cfg, o_probs, o_logq)
        tol_p = nf.tol(1e-9, fl_p)
        near = (np.abs(u - o_probs) < tol_p).any(axis=(1, 2))      # chains with a draw too close to call
        n_near += int((np.abs(u - o_probs) < 1e-9).sum())
        ok = ~near
        assert ok.sum() >= 0.9 * n_s
        assert (cfg[d][ok] == o_cfg[ok]).all()
        assert np.abs(probs[d][ok] - o_probs[ok]).max() < tol_p
        assert np.abs(logq[d][ok] - o_logq[ok]).max() < nf.tol(1e-9 * max(1.0, np.abs(o_logq).max()), fl_q)
        assert (E[d][ok] == exact.energy(o_cfg[ok], Jr[d], Jd[d])).all()
    assert flags["near_threshold"] >= n_near
    assert flags["rho_zero"] == 0 and flags["nonfinite"] == 0


def test_teacher_forcing_normalisation(tn):
    """Pin 7 on the GPU path: sum over all 2^16 configurations of q(s) = 1 at 4x4, chi = 2."""
    L, chi, beta = 4, 2, 1.0
    Jr, Jd = make_couplings(L, 1, 31)
    cfgs = exact.all_configs(L)                     # (65536, 4, 4)
    n = cfgs.shape[0]
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n)
    ctx.tnmc_build_envs()
    forced = torch.from_numpy(pack(cfgs[None]).view(np.int32)).cuda()
    bits, logq = ctx.tnmc_sample(n, 1, forced_cfg_bits=forced)
    assert (bits == forced).all()
    total = np.exp(logq.cpu().numpy()).sum()
    assert abs(total - 1.0) < 1e-10
    cache, _ = bmps.build_cache(Jr[0], Jd[0], beta, chi)
    idx = np.arange(0, n, 97)
    _, o_logq, _ = sampler.sample(cache, Jd[0], beta, np.zeros((len(idx), L, L)), forced=cfgs[idx])
    assert np.abs(logq.cpu().numpy()[0, idx] - o_logq).max() < 1e-9
