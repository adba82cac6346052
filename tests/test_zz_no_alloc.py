"""tnmc_observables_static (the entry point that allocates nothing: magnetisation scratch in a static device
array of the library) against tnmc_observables on the same inputs, bit-exactly (integer sums), on two calls in a
row -- the second call reuses the array with the first call's contents still in it -- and the size limit.
Collected last (file name) so that a failure here hides no other test under `pytest -x`."""
import numpy as np
import pytest

from tnmc_workloads import make_couplings

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def test_observables_static_matches_observables_twice():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2509_19006_b200 import tnmc
    dev = torch.device("cuda:0")
    prev = None
    for call, (L, chi, beta, n_dis, n_s) in enumerate([(33, 4, 0.8, 3, 150), (12, 3, 1.5, 2, 97)]):
        Jr, Jd = make_couplings(L, n_dis, 900 + L)
        ctx = tnmc.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_s)
        ctx.tnmc_build_envs()
        bits, logq = ctx.tnmc_sample(n_s, 5)
        E = ctx.tnmc_energy(bits)
        acc, _, _, _ = ctx.tnmc_metropolis(E, logq, 5)
        _, ref_state, ref_sums = ctx.tnmc_observables(bits, E, acc)
        state = (torch.zeros(n_dis, dtype=torch.int32, device=dev), torch.zeros(n_dis, dtype=torch.int32, device=dev))
        sums = torch.zeros((n_dis, 5), dtype=torch.float64, device=dev)
        before = torch.cuda.memory_allocated()
        ctx.tnmc_observables_static(bits, E, acc, state, sums)
        assert torch.cuda.memory_allocated() == before
        torch.cuda.synchronize()
        assert torch.equal(sums, ref_sums), (call, sums, ref_sums)
        assert torch.equal(state[0], ref_state[0]) and torch.equal(state[1], ref_state[1])
        assert float(sums[:, 4].min()) >= 0 and bool((sums[:, 1] > 0).all())      # not vacuous: sums are populated
        if prev is not None:
            assert not torch.equal(sums[: prev.shape[0]], prev[: sums.shape[0]])  # the second call is a different case
        prev = sums.clone()
    # beyond the static array: a clear error, nothing launched
    cap = int(tnmc.lib.tnmc_observables_static_max())
    assert cap == 1 << 20
    n_big = cap // n_dis + 1
    ctx_big = tnmc.Context(L, chi, beta, torch.from_numpy(Jr).to(dev), torch.from_numpy(Jd).to(dev), n_big)
    z8 = torch.zeros((n_dis, n_big), dtype=torch.uint8, device=dev)
    z32 = torch.zeros((n_dis, n_big), dtype=torch.int32, device=dev)
    zb = torch.zeros((n_dis, n_big, L, 1), dtype=torch.int32, device=dev)
    with pytest.raises(tnmc.TnmcError) as ei:
        ctx_big.tnmc_observables_static(zb, z32, z8, state, sums)
    assert ei.value.status == tnmc.TNMC_EINVAL and "exceeds the static scratch" in str(ei.value)
