"""GPU parity of the fused sampling pass (tnmc_sample_fused: E and M accumulated inside the left sweep, configurations
optional) and of tnmc_replica_overlap, against oracle/exact.py, oracle/observables.py and the standalone kernels.
Everything compared here is an integer: bit-exact."""
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


# lattice widths around the 32-bit word: one ragged word, exactly one / two words (bond across the word boundary), ragged second and third word
@pytest.mark.parametrize("L,chi,beta,n_dis,n_s,ckpt,prec", [
    (6, 2, 1.0, 3, 70, 0, 0), (32, 3, 0.7, 2, 130, 0, 0), (33, 4, 0.8, 2, 150, 0, 0), (64, 3, 0.6, 2, 40, 0, 0),
    (70, 4, 0.9, 2, 33, 0, 0), (33, 4, 0.8, 2, 150, 5, 0), (70, 3, 0.9, 1, 140, 16, 0), (33, 8, 0.8, 2, 60, 0, 1), (40, 16, 1.0, 1, 50, 7, 2)])
def test_sample_fused_parity(tn, L, chi, beta, n_dis, n_s, ckpt, prec):
    dev = torch.device("cuda:0")
    Jr, Jd = make_couplings(L, n_dis, 700 + L)
    Jr[:, ::3, ::4] = 0                                       # some diluted bonds
    Jd[:, 1::4, ::3] = 0
    Jr[:, :, L - 1] = 0
    Jd[:, L - 1, :] = 0
    ctx = tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s, ckpt_stride=ckpt, prec=prec)
    ctx.tnmc_build_envs()
    bits0, logq0 = ctx.tnmc_sample(n_s, 9)
    E0 = ctx.tnmc_energy(bits0)
    bits1, logq1, E1, M1 = ctx.tnmc_sample_fused(n_s, 9)
    assert torch.equal(bits1, bits0) and torch.equal(logq1, logq0)
    assert torch.equal(E1, E0)
    cfg = unpack(bits0.cpu().numpy().view(np.uint32), L)
    for d in range(n_dis):
        assert (E1[d].cpu().numpy() == exact.energy(cfg[d], Jr[d], Jd[d])).all()
        assert (M1[d].cpu().numpy() == observables.magnetisation(cfg[d])).all()
    # configurations not kept: same E, M, log q (in checkpoint mode the last row of a segment travels through the carry buffer)
    none, logq2, E2, M2 = ctx.tnmc_sample_fused(n_s, 9, keep_cfg=False)
    assert none is None and torch.equal(logq2, logq0) and torch.equal(E2, E0) and torch.equal(M2, M1)
    # a sub-range of disorders and a sample offset
    if n_dis > 1:
        _, lq3, E3, M3 = ctx.tnmc_sample_fused(n_s // 2, 9, sample_offset=3, dis_begin=1, dis_count=1, keep_cfg=False)
        b4, lq4 = ctx.tnmc_sample(n_s // 2, 9, sample_offset=3, dis_begin=1, dis_count=1)
        assert torch.equal(lq3, lq4) and torch.equal(E3, ctx.tnmc_energy(b4, dis_begin=1))


def test_sample_fused_refuses_real_couplings(tn):
    dev = torch.device("cuda:0")
    L = 8
    Jr, Jd = make_couplings(L, 1, 5)
    ctx = tn.Context(L, 4, 1.0, torch.from_numpy(Jr.astype(np.float64)).to(dev), torch.from_numpy(Jd.astype(np.float64)).to(dev), 4)
    ctx.tnmc_build_envs()
    with pytest.raises(tn.TnmcError) as ei:
        ctx.tnmc_sample_fused(4, 1)
    assert ei.value.status == tn.TNMC_ESTATE


@pytest.mark.parametrize("L,chi,beta,n_dis,n_s", [(6, 2, 1.2, 3, 200), (33, 3, 1.0, 2, 150), (64, 2, 0.9, 2, 97)])
def test_replica_overlap_parity(tn, L, chi, beta, n_dis, n_s):
    dev = torch.device("cuda:0")
    Jr, Jd = make_couplings(L, n_dis, 800 + L)
    ctx = tn.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s)
    ctx.tnmc_build_envs()
    reps = []
    for seed in (21, 22):                                     # two independent replicas: different Philox keys
        bits, logq = ctx.tnmc_sample(n_s, seed)
        E = ctx.tnmc_energy(bits)
        acc, n_acc, _, _ = ctx.tnmc_metropolis(E, logq, seed)
        assert 0 < int(n_acc.sum()) < n_dis * (n_s - 1)       # truncated chi: some proposals are rejected
        reps.append((bits, acc))
    (ba, aa), (bb, ab) = reps
    q, state, sums = ctx.tnmc_replica_overlap(ba, aa, bb, ab)
    ca, cb = unpack(ba.cpu().numpy().view(np.uint32), L), unpack(bb.cpu().numpy().view(np.uint32), L)
    aa_h, ab_h = aa.cpu().numpy(), ab.cpu().numpy()
    for d in range(n_dis):
        oq, os_, cur_a, cur_b = observables.replica_overlap(ca[d], aa_h[d], cb[d], ab_h[d])
        assert (q[d].cpu().numpy() == oq).all()
        assert [int(v) for v in sums[d].cpu().numpy()] == os_
        assert (unpack(state[0].cpu().numpy().view(np.uint32), L)[d] == cur_a).all()
        assert (unpack(state[1].cpu().numpy().view(np.uint32), L)[d] == cur_b).all()
    # two chunks with the carried states give the same steps and sums
    h = n_s // 3
    cut = lambda t, lo, hi: t[:, lo:hi].contiguous()
    q1, st, sm = ctx.tnmc_replica_overlap(cut(ba, 0, h), cut(aa, 0, h), cut(bb, 0, h), cut(ab, 0, h))
    q2, st, sm = ctx.tnmc_replica_overlap(cut(ba, h, n_s), cut(aa, h, n_s), cut(bb, h, n_s), cut(ab, h, n_s), state=st, sums=sm)
    assert torch.equal(torch.cat([q1, q2], dim=1), q) and torch.equal(sm, sums)
    assert torch.equal(st[0], state[0]) and torch.equal(st[1], state[1])
    # a replica against itself: q = N at every step
    qs, _, _ = ctx.tnmc_replica_overlap(ba, aa, ba, aa)
    assert bool((qs == L * L).all())
