"""GPU parity, second part: Metropolis scan, checkpoint/recompute policy, chunked calls, the
host-buffer entry point, and a subset of config C2 (32x32, chi=16, three betas)."""
import numpy as np
import pytest

from oracle import bmps, exact, metropolis, philox, sampler
from tnmc_workloads import CONFIGS, make_couplings

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


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def test_metropolis_parity(tn):
    """Eq. 10 scan against the oracle on synthetic (E, log q) streams, in two chunks."""
    rng = np.random.default_rng(5)
    n_dis, n_s, beta, seed, first = 7, 300, 0.9, 4242, 11
    E = rng.integers(-40, 40, (n_dis, n_s)).astype(np.int32)
    logq = -0.9 * E + rng.normal(0, 1.5, (n_dis, n_s))
    L = 4
    Jr, Jd = make_couplings(L, n_dis, 1)
    ctx = _ctx(tn, L, 2, beta, Jr, Jd, 4, first_disorder=first)
    Et, qt = torch.from_numpy(E).cuda(), torch.from_numpy(logq).cuda()
    h = 120
    acc1, n1, state, s1 = ctx.tnmc_metropolis(Et[:, :h].contiguous(), qt[:, :h].contiguous(), seed, want_sum_min1=True)
    acc2, n2, state, s2 = ctx.tnmc_metropolis(Et[:, h:].contiguous(), qt[:, h:].contiguous(), seed, step_offset=h,
                                              state=state, want_sum_min1=True)
    acc = torch.cat([acc1, acc2], dim=1).cpu().numpy()
    for d in range(n_dis):
        u = philox.metropolis_uniforms(seed, first + d, np.arange(n_s))
        o_acc, o_n, cE, cq, ci, sm = metropolis.metropolis_scan(E[d], logq[d], beta, u)
        assert (acc[d] == o_acc).all()
        assert int(n1[d] + n2[d]) == o_n
        assert int(state[1][d]) == cE and int(state[2][d]) == ci
        assert float(state[0][d]) == cq
        assert abs(float(s1[d] + s2[d]) - sm) < 1e-9 * max(1.0, sm)


def test_exact_chi_acceptance_is_one(tn):
    """north_star: chi >= 2^(L/2) => log q(s) = -beta E(s) - log Z and every proposal is accepted (C1)."""
    cfgC = CONFIGS["C1"]
    L, chi, beta, n_dis, n_s = cfgC["L"], cfgC["chi"], cfgC["betas"][0], cfgC["n_dis"], cfgC["n_samples"]
    Jr, Jd = make_couplings(L, n_dis, cfgC["inst_seed"])
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, cfgC["seed"])
    E = ctx.tnmc_energy(bits)
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, cfgC["seed"])
    resid = logq + beta * E.double() + logZ[:, None]
    assert resid.abs().max().item() < 1e-9
    # log A = resid differences ~ 1e-12; acceptance needs log u < log A, true unless u ~ 1
    assert (n_acc == n_s - 1).all()
    for d in range(n_dis):
        assert abs(logZ[d].item() - exact.transfer_logZ(Jr[d], Jd[d], beta)) < 1e-10 * abs(logZ[d].item())


@pytest.mark.parametrize("L,chi,k", [(12, 4, 3), (12, 4, 5), (9, 4, 1), (10, 8, 4), (8, 4, 7), (20, 16, 6), (26, 32, 7)])
def test_checkpoint_recompute_matches_full_stack(tn, L, chi, k):
    """a-6: the checkpoint + segment-recompute policy gives bit-identical samples and log q."""
    n_dis, n_s, beta, seed = 3, 37, 1.0, 99
    Jr, Jd = make_couplings(L, n_dis, 500 + L)
    full = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    lz_f = full.tnmc_build_envs()
    b_f, q_f = full.tnmc_sample(n_s, seed)
    ck = _ctx(tn, L, chi, beta, Jr, Jd, n_s, ckpt_stride=k)
    lz_c = ck.tnmc_build_envs()
    b_c, q_c = ck.tnmc_sample(n_s, seed)
    assert torch.equal(lz_f, lz_c)
    assert torch.equal(b_f, b_c)
    assert torch.equal(q_f, q_c)
    # a checkpoint row can be read back, a recomputed one cannot
    ck.tnmc_get_env_row(0, 0)
    if k > 1 and L - 1 != 1:
        with pytest.raises(tn.TnmcError) as ei:
            ck.tnmc_get_env_row(0, 1)
        assert ei.value.status == tn.TNMC_ESTATE


def test_chunked_calls_are_consistent(tn):
    """Philox indexing by (disorder, sample, site): chunking over disorders / samples changes nothing."""
    L, chi, beta, n_dis, n_s, seed = 10, 4, 1.0, 4, 150, 7
    Jr, Jd = make_couplings(L, n_dis, 321)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    ctx.tnmc_build_envs()
    b_all, q_all = ctx.tnmc_sample(n_s, seed)
    b_d, q_d = ctx.tnmc_sample(n_s, seed, dis_begin=2, dis_count=2)
    assert torch.equal(b_all[2:], b_d) and torch.equal(q_all[2:], q_d)
    b_s, q_s = ctx.tnmc_sample(50, seed, sample_offset=100)
    assert torch.equal(b_all[:, 100:150], b_s) and torch.equal(q_all[:, 100:150], q_s)
    # a context that only knows disorders 2..3 (first_disorder = 2) reproduces them
    sub = _ctx(tn, L, chi, beta, Jr[2:], Jd[2:], n_s, first_disorder=2)
    sub.tnmc_build_envs()
    b2, q2 = sub.tnmc_sample(n_s, seed)
    assert torch.equal(b_all[2:], b2) and torch.equal(q_all[2:], q2)


def test_run_host_matches_device_calls(tn):
    L, chi, beta, n_dis, n_s, seed = 12, 8, 1.0, 3, 40, 17
    Jr, Jd = make_couplings(L, n_dis, 654)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, seed)
    E = ctx.tnmc_energy(bits)
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, seed)
    ws = torch.empty(tn.tnmc_run_host_workspace_bytes(L, chi, n_dis, n_s), dtype=torch.uint8, device="cuda")
    out = tn.tnmc_run_host(L, chi, beta, torch.from_numpy(Jr).pin_memory(), torch.from_numpy(Jd).pin_memory(), n_s, seed, ws)
    assert torch.equal(out["cfg_bits"], bits.cpu()) and torch.equal(out["E"], E.cpu())
    assert torch.equal(out["logq"], logq.cpu()) and torch.equal(out["accepted"], acc.cpu())
    assert torch.equal(out["logZ"], logZ.cpu()) and torch.equal(out["n_accepted"], n_acc.cpu())


def test_error_paths(tn):
    L = 6
    Jr, Jd = make_couplings(L, 2, 1)
    ctx = _ctx(tn, L, 4, 1.0, Jr, Jd, 8)
    with pytest.raises(tn.TnmcError) as ei:
        ctx.tnmc_sample(8, 1)
    assert ei.value.status == tn.TNMC_ESTATE
    ctx.tnmc_build_envs()
    with pytest.raises(tn.TnmcError) as ei:
        ctx.tnmc_sample(9, 1)
    assert ei.value.status == tn.TNMC_EINVAL
    with pytest.raises(tn.TnmcError) as ei:
        ctx.tnmc_sample(8, 1, dis_begin=1, dis_count=2)
    assert ei.value.status == tn.TNMC_EINVAL
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(tn.TnmcError) as ei:
        tn.Context(L, 4, 1.0, torch.from_numpy(Jr).cuda(), torch.from_numpy(Jd).cuda(), 8, workspace=small)
    assert ei.value.status == tn.TNMC_ENOMEM
    with pytest.raises(tn.TnmcError):
        tn.Context(L, 64, 1.0, torch.from_numpy(Jr).cuda(), torch.from_numpy(Jd).cuda(), 8)


@pytest.mark.parametrize("beta", CONFIGS["C2"]["betas"])
def test_config_c2_subset(tn, beta):
    """Config C2 (32x32, chi=16, 100 x 100) on the GPU in full; the oracle checks disorders 0, 57, 99
    x 24 samples (the oracle's sampler costs ~1 s per disorder at this size)."""
    c = CONFIGS["C2"]
    L, chi, n_dis, n_s = c["L"], c["chi"], c["n_dis"], c["n_samples"]
    Jr, Jd = make_couplings(L, n_dis, c["inst_seed"])
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs().cpu().numpy()
    probs = torch.zeros((n_dis, n_s, L, L), dtype=torch.float64, device="cuda")
    bits, logq = ctx.tnmc_sample(n_s, c["seed"], probs=probs)
    E = ctx.tnmc_energy(bits).cpu().numpy()
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["rho_zero"] == 0
    cfg = unpack(_u32(bits), L)
    n_chk = 24
    for d in (0, 57, 99):
        cache, ls = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        cache_p, ls_p = nf.perturbed_cache(Jr[d], Jd[d], beta, chi)
        lz, _ = bmps.log_z(cache[0], ls[0])
        assert abs(logZ[d] - lz) <= nf.tol(1e-10 * abs(lz), nf.logz_floor(cache, ls, cache_p, ls_p))
        u = np.empty((n_chk, L, L))
        for r in range(L):
            for cc in range(L):
                u[:, r, cc] = philox.spin_uniforms(c["seed"], d, np.arange(n_chk), r * L + cc)
        o_cfg, o_logq, o_probs = sampler.sample(cache, Jd[d], beta, u)
        p_gpu = probs[d, :n_chk].cpu().numpy()
        fl_p, fl_q = nf.probs_floor(cache_p, Jd[d], beta, o_cfg, o_probs, o_logq)
        tol_p = nf.tol(1e-9, fl_p)
        same = (cfg[d, :n_chk] == o_cfg).all(axis=(1, 2))
        near = (np.abs(u - o_probs) < tol_p).any(axis=(1, 2))
        assert (same | near).all()
        ok = same & ~near
        assert ok.sum() >= n_chk - 2
        assert np.abs(p_gpu[ok] - o_probs[ok]).max() < tol_p
        assert np.abs(logq[d, :n_chk].cpu().numpy()[ok] - o_logq[ok]).max() < nf.tol(1e-9 * np.abs(o_logq).max(), fl_q)
        assert (E[d, :n_chk][ok] == exact.energy(o_cfg[ok], Jr[d], Jd[d])).all()


@pytest.mark.parametrize("L,chi,n_dis,n_s", [(2, 2, 1, 1), (3, 32, 2, 2), (5, 32, 1, 129), (2, 32, 3, 1)])
def test_degenerate_sizes(tn, L, chi, n_dis, n_s):
    """smallest lattice, one sample, chi far above the exact bound (the padded-bond code paths with tiny bonds),
    one chain more than a tile: exact chi, so log q = -beta E - log Z and log Z = brute force."""
    beta, seed = 0.9, 3
    Jr, Jd = make_couplings(L, n_dis, 70 + L)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, seed)
    E = ctx.tnmc_energy(bits)
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, seed)
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["rho_zero"] == 0 and flags["logz_nonpos"] == 0
    for d in range(n_dis):
        _, _, lz, _ = exact.brute_force(Jr[d], Jd[d], beta)
        assert abs(logZ[d].item() - lz) < 1e-10 * abs(lz)
    assert (logq + beta * E.double() + logZ[:, None]).abs().max().item() < 1e-9
    assert (n_acc == n_s - 1).all() and (acc[:, 0] == 1).all()
    cfg = unpack(_u32(bits), L)
    for d in range(n_dis):
        assert (E[d].cpu().numpy() == exact.energy(cfg[d], Jr[d], Jd[d])).all()
