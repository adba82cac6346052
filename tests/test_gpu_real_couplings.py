"""GPU parity for real-valued couplings (Gaussian EA; tnmc_create_real / tnmc_energy_real /
tnmc_metropolis_real) against the oracle: log Z (rel 1e-10), conditionals (abs 1e-9), spins bit-exact off the
near-threshold chains, log q, energies (floating point: 1e-12 of sum |J|), the Metropolis scan, the exact-chi
limit, checkpoint mode, and the reduced-precision mode's invariants."""
import numpy as np
import pytest

from oracle import bmps, exact, metropolis, observables, philox, sampler
from tnmc_workloads import make_gaussian_couplings

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


def _ctx(tn, L, chi, beta, Jr, Jd, n_s, **kw):
    dev = torch.device("cuda:0")
    return tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s, **kw)


@pytest.mark.parametrize("L,chi,beta,n_dis,n_s,k", [(6, 8, 0.9, 2, 40, 0), (12, 8, 1.0, 2, 30, 0), (33, 8, 0.7, 1, 20, 0),
                                                    (20, 20, 1.2, 1, 140, 0), (12, 4, 1.0, 2, 30, 5)])
def test_real_couplings_parity(tn, L, chi, beta, n_dis, n_s, k):
    seed, first = 17, 3
    Jr, Jd = make_gaussian_couplings(L, n_dis, 50 + L)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s, first_disorder=first, ckpt_stride=k)
    logZ = ctx.tnmc_build_envs().cpu().numpy()
    probs = torch.zeros((n_dis, n_s, L, L), dtype=torch.float64, device="cuda")
    bits, logq = ctx.tnmc_sample(n_s, seed, probs=probs)
    E = ctx.tnmc_energy(bits)
    assert E.dtype == torch.float64
    acc, n_acc, state, smin = ctx.tnmc_metropolis(E, logq, seed, want_sum_min1=True)
    flags = ctx.tnmc_get_flags()
    assert flags["nonfinite"] == 0 and flags["jacobi_limit"] == 0 and flags["rho_zero"] == 0 and flags["logz_nonpos"] == 0
    cfg = unpack(bits.cpu().numpy().view(np.uint32), L)
    E_h, q_h, acc_h = E.cpu().numpy(), logq.cpu().numpy(), acc.cpu().numpy()
    for d in range(n_dis):
        cache, ls = bmps.build_cache(Jr[d], Jd[d], beta, chi)
        cache_p, ls_p = nf.perturbed_cache(Jr[d], Jd[d], beta, chi)
        lz, sign = bmps.log_z(cache[0], ls[0])
        assert sign == 1.0
        assert abs(logZ[d] - lz) <= nf.tol(1e-10 * abs(lz), nf.logz_floor(cache, ls, cache_p, ls_p))
        u = np.empty((n_s, L, L))
        for r in range(L):
            for c in range(L):
                u[:, r, c] = philox.spin_uniforms(seed, first + d, np.arange(n_s), r * L + c)
        o_cfg, o_logq, o_probs = sampler.sample(cache, Jd[d], beta, u)
        fl_p, fl_q = nf.probs_floor(cache_p, Jd[d], beta, o_cfg, o_probs, o_logq)
        tol_p = nf.tol(1e-9, fl_p)
        same = (cfg[d] == o_cfg).all(axis=(1, 2))
        near = (np.abs(u - o_probs) < tol_p).any(axis=(1, 2))
        assert (same | near).all()
        ok = same & ~near
        assert ok.sum() >= 0.9 * n_s
        assert np.abs(probs[d].cpu().numpy()[ok] - o_probs[ok]).max() < tol_p
        assert np.abs(q_h[d][ok] - o_logq[ok]).max() < nf.tol(1e-9 * np.abs(o_logq).max(), fl_q)
        # energies of the GPU's own configurations (every chain), floating point
        oE = exact.energy_real(cfg[d], Jr[d], Jd[d])
        scale = np.abs(Jr[d]).sum() + np.abs(Jd[d]).sum()
        assert np.abs(E_h[d] - oE).max() <= 1e-12 * scale
        # Metropolis scan on the GPU's own (E, log q)
        um = philox.metropolis_uniforms(seed, first + d, np.arange(n_s))
        o_acc, o_n, cE, cq, ci, sm = metropolis.metropolis_scan_real(E_h[d], q_h[d], beta, um)
        assert (acc_h[d] == o_acc).all() and int(n_acc[d]) == o_n
        assert float(state[1][d]) == cE and int(state[2][d]) == ci
        assert abs(float(smin[d]) - sm) < 1e-9 * max(1.0, sm)
    # observables along the chain with real energies
    M, st_o, sums = ctx.tnmc_observables(bits, E, acc)
    M_h, sums_h = M.cpu().numpy(), sums.cpu().numpy()
    for d in range(n_dis):
        assert (M_h[d] == observables.magnetisation(cfg[d])).all()
        so, cE, cM = observables.chain_sums_real(E_h[d], M_h[d], acc_h[d])
        assert np.allclose(sums_h[d], so, rtol=1e-12, atol=1e-9)
        assert float(st_o[0][d]) == cE and int(st_o[1][d]) == cM


def test_real_couplings_exact_chi_and_f32_invariants(tn):
    L, chi, beta, n_dis, n_s = 8, 16, 0.8, 2, 64
    Jr, Jd = make_gaussian_couplings(L, n_dis, 99)
    ctx = _ctx(tn, L, chi, beta, Jr, Jd, n_s)
    logZ = ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, 5)
    E = ctx.tnmc_energy(bits)
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, 5)
    assert (logq + beta * E + logZ[:, None]).abs().max().item() < 1e-9
    assert (n_acc == n_s - 1).all()
    for d in range(n_dis):
        assert abs(logZ[d].item() - exact.transfer_logZ(Jr[d], Jd[d], beta)) < 1e-10 * abs(logZ[d].item())
    # wrong entry point for this context
    with pytest.raises(tn.TnmcError) as ei:
        tn._check(tn.lib.tnmc_energy(ctx.h, 0, n_dis, n_s, tn._ptr(bits, torch.int32),
                                     tn._ptr(torch.empty((n_dis, n_s), dtype=torch.int32, device="cuda"), torch.int32)), ctx.h)
    assert ei.value.status == tn.TNMC_ESTATE
    # reduced precision: q normalised, log q consistent with teacher forcing, log Z close
    L2, chi2 = 4, 2
    Jr2, Jd2 = make_gaussian_couplings(L2, 1, 7)
    cfgs = exact.all_configs(L2)
    c32 = _ctx(tn, L2, chi2, 1.0, Jr2, Jd2, cfgs.shape[0], prec=tn.TNMC_F32_LOGSCALE)
    lz32 = c32.tnmc_build_envs()
    forced = torch.from_numpy(pack(cfgs[None]).view(np.int32)).cuda()
    _, lq = c32.tnmc_sample(cfgs.shape[0], 1, forced_cfg_bits=forced)
    assert abs(np.exp(lq.cpu().numpy()).sum() - 1.0) < 1e-10
    cache, ls = bmps.build_cache(Jr2[0], Jd2[0], 1.0, chi2)
    assert abs(lz32[0].item() - bmps.log_z(cache[0], ls[0])[0]) < 1e-4 * abs(lz32[0].item())
