"""GPU parity of tnmc_observables (thermal averages along the Metropolis chain, reading G19) against
oracle/observables.py: magnetisations and the five chain sums are integers -- compared bit-exactly --
on the GPU's own (cfg, E, accepted), in one call and in two chunks with the chain state carried."""
import numpy as np
import pytest

from oracle import exact, observables
from tnmc_workloads import make_couplings

from bitpack import unpack

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tn():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2509_19006_b200 import tnmc
    return tnmc


@pytest.mark.parametrize("L,chi,beta,n_dis,n_s", [(6, 2, 1.0, 3, 200), (33, 4, 0.8, 2, 150), (12, 3, 1.5, 2, 97)])
def test_observables_parity(tn, L, chi, beta, n_dis, n_s):
    dev = torch.device("cuda:0")
    Jr, Jd = make_couplings(L, n_dis, 640 + L)
    ctx = tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s)
    ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(n_s, 11)
    E = ctx.tnmc_energy(bits)
    acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, 11)
    M, state, sums = ctx.tnmc_observables(bits, E, acc)
    cfg = unpack(bits.cpu().numpy().view(np.uint32), L)
    E_h, acc_h, M_h = E.cpu().numpy(), acc.cpu().numpy(), M.cpu().numpy()
    assert 0 < int(n_acc.sum()) < n_dis * (n_s - 1)          # truncated chi: some proposals are rejected
    for d in range(n_dis):
        assert (M_h[d] == observables.magnetisation(cfg[d])).all()
        assert (E_h[d] == exact.energy(cfg[d], Jr[d], Jd[d])).all()
        s, cE, cM = observables.chain_sums(E_h[d], M_h[d], acc_h[d])
        assert [int(v) for v in sums[d].cpu().numpy()] == s
        assert int(state[0][d]) == cE and int(state[1][d]) == cM
    # two chunks with carried state give the same sums
    h = n_s // 3
    _, st, sm = ctx.tnmc_observables(bits[:, :h].contiguous(), E[:, :h].contiguous(), acc[:, :h].contiguous())
    _, st, sm = ctx.tnmc_observables(bits[:, h:].contiguous(), E[:, h:].contiguous(), acc[:, h:].contiguous(), state=st, sums=sm)
    assert torch.equal(sm, sums) and torch.equal(st[0], state[0]) and torch.equal(st[1], state[1])
    # a sub-range of disorders
    _, _, s1 = ctx.tnmc_observables(bits[1:].contiguous(), E[1:].contiguous(), acc[1:].contiguous(), dis_begin=1)
    assert torch.equal(s1, sums[1:])
