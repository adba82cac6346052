"""Contract of the C ABI that include/tnmc.h states beyond the arithmetic: tnmc_create does not wait for the
stream; couplings stored across the open boundary are ignored (energies stay consistent with q); the 32-bit
Philox index words are range-checked."""
import time

import numpy as np
import pytest

from oracle import exact
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


def test_create_does_not_block(tn):
    dev = torch.device("cuda:0")
    L, chi, n_dis = 16, 4, 2
    Jr, Jd = make_couplings(L, n_dis, 77)
    Jr, Jd = torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev)
    ws = torch.empty(tn.tnmc_workspace_bytes(L, chi, n_dis, 8), dtype=torch.uint8, device=dev)
    tn.Context(L, chi, 1.0, Jr, Jd, 8, workspace=ws).close()          # warm: module load, first launch
    torch.cuda.synchronize()
    torch.cuda._sleep(int(0.4 * 1.9e9))                                # ~0.4 s of busy-wait on the current stream
    t0 = time.perf_counter()
    ctx = tn.Context(L, chi, 1.0, Jr, Jd, 8, workspace=ws)
    t_create = time.perf_counter() - t0
    torch.cuda.synchronize()
    t_all = time.perf_counter() - t0
    assert t_all > 0.15, "the sleep kernel did not hold the stream: the test proves nothing"
    assert t_create < 0.05, f"tnmc_create waited for the stream ({t_create:.3f} s of {t_all:.3f} s)"
    logZ = ctx.tnmc_build_envs()
    assert torch.isfinite(logZ).all()


def test_boundary_couplings_are_ignored(tn):
    """Jr at c = L-1 and Jd at r = L-1 name bonds that do not exist: garbage there changes nothing."""
    dev = torch.device("cuda:0")
    L, chi, n_dis, n_s = 33, 4, 2, 40
    Jr, Jd = make_couplings(L, n_dis, 78)
    Jr2, Jd2 = Jr.copy(), Jd.copy()
    Jr2[:, :, L - 1] = -1
    Jd2[:, L - 1, :] = 1
    out = []
    for a, b in ((Jr, Jd), (Jr2, Jd2)):
        ctx = tn.Context(L, chi, 0.9, torch.from_numpy(a).to(dev), torch.from_numpy(b).to(dev), n_s)
        lz = ctx.tnmc_build_envs()
        bits, logq = ctx.tnmc_sample(n_s, 3)
        E = ctx.tnmc_energy(bits)
        out.append((lz.cpu(), bits.cpu(), logq.cpu(), E.cpu()))
    for x, y in zip(*out):
        assert torch.equal(x, y)
    cfg = unpack(out[0][1].numpy().view(np.uint32), L)
    for d in range(n_dis):
        assert (out[1][3][d].numpy() == exact.energy(cfg[d], Jr[d], Jd[d])).all()
    # real couplings: the same rule in energy_real_kernel
    Jrr, Jdr = Jr.astype(np.float64) * 0.7, Jd.astype(np.float64) * 1.3
    Jrr2, Jdr2 = Jrr.copy(), Jdr.copy()
    Jrr2[:, :, L - 1] = 5.0
    Jdr2[:, L - 1, :] = -4.0
    Es = []
    for a, b in ((Jrr, Jdr), (Jrr2, Jdr2)):
        ctx = tn.Context(L, chi, 0.9, torch.from_numpy(a).to(dev), torch.from_numpy(b).to(dev), n_s)
        Es.append(ctx.tnmc_energy(out[0][1].to(dev)).cpu())
    assert torch.equal(Es[0], Es[1])


def test_philox_index_words_are_range_checked(tn):
    dev = torch.device("cuda:0")
    L, chi = 8, 4
    Jr, Jd = make_couplings(L, 1, 79)
    ctx = tn.Context(L, chi, 1.0, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), 4)
    ctx.tnmc_build_envs()
    bits, logq = ctx.tnmc_sample(4, 1, sample_offset=(1 << 32) - 4)          # the last four indices are fine
    with pytest.raises(tn.TnmcError) as ei:
        ctx.tnmc_sample(4, 1, sample_offset=(1 << 32) - 3)
    assert ei.value.status == tn.TNMC_EINVAL and "2^32" in str(ei.value)
    E = ctx.tnmc_energy(bits)
    ctx.tnmc_metropolis(E, logq, 1, step_offset=(1 << 32) - 4)
    with pytest.raises(tn.TnmcError):
        ctx.tnmc_metropolis(E, logq, 1, step_offset=(1 << 32) - 3)
