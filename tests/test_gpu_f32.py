"""GPU tests of the reduced-precision mode TNMC_F32_LOGSCALE (environment stack stored in FP32).
north_star tolerance for a reduced-precision path: log Z relative 1e-4 against the oracle; spins are not
expected to be bit-identical.  What must hold exactly in any precision: q is a normalised distribution
(sum over all configurations = 1), log q returned with a sample is the log of the probabilities used to
draw it (teacher forcing reproduces it bit for bit) -- that is what keeps the Metropolis correction exact."""
import numpy as np
import pytest

from oracle import bmps, exact
from tnmc_workloads import CONFIGS, make_couplings

from bitpack import pack, unpack

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tn():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2509_19006_b200 import tnmc
    return tnmc


def _ctx(tn, L, chi, beta, Jr, Jd, n_s, **kw):
    dev = torch.device("cuda:0")
    return tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s, **kw)


@pytest.mark.parametrize("mode", ["x3", "fast"])
@pytest.mark.parametrize("L,chi,beta,k", [(8, 4, 1.0, 0), (12, 8, 1.0, 0), (24, 32, 1.0, 0), (32, 16, 2.0, 0), (12, 8, 1.0, 4)])
def test_f32_logz_and_consistency(tn, L, chi, beta, k, mode):
    n_dis, n_s, seed = 2, 40, 9
    Jr, Jd = make_couplings(L, n_dis, 900 + L)
    prec = tn.TNMC_F32_LOGSCALE if mode == "x3" else tn.TNMC_TF32_FAST
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s, prec=prec, ckpt_stride=k)
    ref = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs().cpu().numpy()
    logZ64 = ref.tnmc_build_envs().cpu().numpy()
    probs = torch.zeros((n_dis, n_s, L, L), dtype=torch.float64, device="cuda")
    bits, logq = ctx.tnmc_sample(n_s, seed, probs=probs)
    flags = ctx.tnmc_get_flags()
    # (rho_zero is informational here: at beta = 2 a conditional weight ~1e-10 of the other can round to 0 in FP32)
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["logz_nonpos"] == 0
    for d in range(n_dis):
        cache, ls = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        lz, _ = bmps.log_z(cache[0], ls[0])
        assert abs(logZ[d] - lz) <= 1e-4 * abs(lz)
        assert abs(logZ[d] - logZ64[d]) <= 1e-4 * abs(lz)
    # log q is the log of the probabilities actually used: teacher forcing reproduces it bit for bit,
    # and it equals the sum of the logs of the reported conditionals
    b2, q2 = ctx.tnmc_sample(n_s, seed, forced_cfg_bits=bits)
    assert torch.equal(b2, bits) and torch.equal(q2, logq)
    cfg = unpack(bits.cpu().numpy().view(np.uint32), L)
    p = probs.cpu().numpy()
    lq = np.where(cfg == 1, np.log(p), np.log1p(-p)).sum(axis=(2, 3))
    assert np.abs(lq - logq.cpu().numpy()).max() < 1e-9 * L * L
    # the reduced-precision conditionals stay close to the FP64 path's on the same configurations
    p64 = torch.zeros_like(probs)
    ref.tnmc_sample(n_s, seed, forced_cfg_bits=bits, probs=p64)
    # plain TF32 products: 10-bit mantissa inputs; 3xTF32: FP32-level accuracy
    assert (probs - p64).abs().mean().item() < (5e-3 if mode == "fast" else 2e-5)
    E = ctx.tnmc_energy(bits).cpu().numpy()
    for d in range(n_dis):
        assert (E[d] == exact.energy(cfg[d], Jr[d], Jd[d])).all()


def test_f32_q_is_normalised(tn):
    L, chi, beta = 4, 2, 1.0
    Jr, Jd = make_couplings(L, 1, 31)
    cfgs = exact.all_configs(L)
    n = cfgs.shape[0]
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n, prec=tn.TNMC_F32_LOGSCALE)
    ctx.tnmc_build_envs()
    forced = torch.from_numpy(pack(cfgs[None]).view(np.int32)).cuda()
    _, logq = ctx.tnmc_sample(n, 1, forced_cfg_bits=forced)
    assert abs(np.exp(logq.cpu().numpy()).sum() - 1.0) < 1e-10


@pytest.mark.parametrize("mode", ["x3", "fast"])
def test_f32_exact_chi_residual(tn, mode):
    """C1 (exact chi): log q + beta E + log Z vanishes up to the TF32 rounding of the contractions (10-bit
    mantissa inputs: ~1e-3 per conditional, 64 sites), and nearly every proposal is accepted."""
    c = CONFIGS["C1"]
    L, chi, beta, n_dis, n_s = c["L"], c["chi"], c["betas"][0], c["n_dis"], c["n_samples"]
    Jr, Jd = make_couplings(L, n_dis, c["inst_seed"])
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s, prec=tn.TNMC_F32_LOGSCALE if mode == "x3" else tn.TNMC_TF32_FAST)
    logZ = ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, c["seed"])
    E = ctx.tnmc_energy(bits)
    resid = logq + beta * E.double() + logZ[:, None]
    print(mode, 'exact-chi residual: max', resid.abs().max().item(), 'rms', resid.pow(2).mean().sqrt().item())
    if mode == "fast":
        assert resid.abs().max().item() < 0.2 and resid.pow(2).mean().sqrt().item() < 0.05
    else:
        assert resid.abs().max().item() < 2e-3 and resid.pow(2).mean().sqrt().item() < 5e-4
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, c["seed"])
    assert (n_acc >= 0.8 * n_s).all()
    assert tn.tnmc_workspace_bytes(64, 32, 10, 8, prec=tn.TNMC_F32_LOGSCALE) < tn.tnmc_workspace_bytes(64, 32, 10, 8)


@pytest.mark.parametrize("L,chi,beta,k", [(12, 8, 1.0, 0), (24, 32, 1.0, 0), (32, 16, 2.0, 0), (20, 16, 1.0, 6)])
def test_f32_store_mode(tn, L, chi, beta, k):
    """TNMC_F32_STORE: FP32 stack, all arithmetic FP64.  Conditionals stay within ~1e-5 of the FP64 path (the
    tensors are rounded once per stored row), log Z within 1e-4 of the oracle, q normalised by construction
    (log q = sum of the logs of the reported conditionals, teacher forcing reproduces it bit for bit)."""
    n_dis, n_s, seed = 2, 40, 9
    Jr, Jd = make_couplings(L, n_dis, 900 + L)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s, prec=tn.TNMC_F32_STORE, ckpt_stride=k)
    ref = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs().cpu().numpy()
    ref.tnmc_build_envs()
    probs = torch.zeros((n_dis, n_s, L, L), dtype=torch.float64, device="cuda")
    bits, logq = ctx.tnmc_sample(n_s, seed, probs=probs)
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["logz_nonpos"] == 0 and flags["rho_zero"] == 0
    for d in range(n_dis):
        cache, ls = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        lz, _ = bmps.log_z(cache[0], ls[0])
        assert abs(logZ[d] - lz) <= 1e-4 * abs(lz)
    b2, q2 = ctx.tnmc_sample(n_s, seed, forced_cfg_bits=bits)
    assert torch.equal(b2, bits) and torch.equal(q2, logq)
    cfg = unpack(bits.cpu().numpy().view(np.uint32), L)
    p = probs.cpu().numpy()
    with np.errstate(divide="ignore"):
        lq = np.where(cfg == 1, np.log(p), np.log1p(-p)).sum(axis=(2, 3))
    assert np.abs(lq - logq.cpu().numpy()).max() < 1e-9 * L * L
    p64 = torch.zeros_like(probs)
    _, q64 = ref.tnmc_sample(n_s, seed, forced_cfg_bits=bits, probs=p64)
    assert (probs - p64).abs().mean().item() < 1e-5
    E = ctx.tnmc_energy(bits)
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, seed)
    acc64, n_acc64, _, _ = ref.tnmc_metropolis(E, q64, seed)
    assert abs(int(n_acc.sum()) - int(n_acc64.sum())) <= 0.05 * n_dis * n_s
    assert tn.tnmc_workspace_bytes(64, 32, 10, 8, prec=tn.TNMC_F32_STORE) < tn.tnmc_workspace_bytes(64, 32, 10, 8)
