"""CPU-side checks (no GPU): the C-ABI library loads and exports every symbol include/tnmc.h
declares; argument validation that needs no device; the closed-form bond dimensions used by the
kernels; the algorithmic-work model used by bench.py; the bit packing helper."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2509_19006_b200 import build
    return ctypes.CDLL(build.build())


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "tnmc.h")).read()
    names = sorted(set(re.findall(r"\b(tnmc_[a-z0-9_]+)\s*\(", hdr)))
    assert {"tnmc_create", "tnmc_build_envs", "tnmc_sample", "tnmc_energy", "tnmc_metropolis"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_workspace_bytes_and_argument_errors(lib):
    lib.tnmc_workspace_bytes.restype = ctypes.c_size_t
    lib.tnmc_workspace_bytes.argtypes = [ctypes.c_int] * 6
    assert lib.tnmc_workspace_bytes(1, 4, 1, 1, 0, 0) == 0          # L < 2
    assert lib.tnmc_workspace_bytes(8, 1, 1, 1, 0, 0) == 0          # chi < 2
    assert lib.tnmc_workspace_bytes(8, 33, 1, 1, 0, 0) == 0         # chi > 32
    assert lib.tnmc_workspace_bytes(8, 4, 0, 1, 0, 0) == 0
    assert lib.tnmc_workspace_bytes(8, 4, 1, 1, 4, 0) == 0          # unknown precision
    assert lib.tnmc_workspace_bytes(64, 32, 8, 8, 2, 0) == lib.tnmc_workspace_bytes(64, 32, 8, 8, 1, 0)   # both FP32 stacks
    f64, f32 = lib.tnmc_workspace_bytes(64, 32, 8, 8, 0, 0), lib.tnmc_workspace_bytes(64, 32, 8, 8, 1, 0)
    assert 0 < f32 < f64                                            # TNMC_F32_LOGSCALE halves the stack
    full = lib.tnmc_workspace_bytes(512, 32, 4, 8, 0, 0)
    ck = lib.tnmc_workspace_bytes(512, 32, 4, 8, 0, 23)
    assert 0 < ck < full / 5                                        # checkpointing shrinks the stack
    # the env stack dominates: L rows x L sites x 2 P^2 doubles per disorder
    assert full > 4 * 512 * 512 * 2 * 32 * 32 * 8
    lib.tnmc_create.restype = ctypes.c_int
    h = ctypes.c_void_p()
    st = lib.tnmc_create(ctypes.byref(h), 8, 4, ctypes.c_double(1.0), 1, None, None, ctypes.c_uint64(0), 1, 0, 0, None,
                         ctypes.c_size_t(0), None)
    assert st == 1 and not h.value                                   # TNMC_EINVAL, no context
    lib.tnmc_last_error.restype = ctypes.c_char_p
    assert b"NULL" in lib.tnmc_last_error(None)
    # the Philox counter word of the disorder index is 32 bits: first_disorder + n_dis beyond 2^32 is refused
    # (argument check only: the fake pointers are never dereferenced on this path)
    need = lib.tnmc_workspace_bytes(8, 4, 2, 1, 0, 0)
    fake = ctypes.c_void_p(1 << 20)
    st = lib.tnmc_create(ctypes.byref(h), 8, 4, ctypes.c_double(1.0), 2, fake, fake, ctypes.c_uint64((1 << 32) - 1), 1, 0, 0, fake,
                         ctypes.c_size_t(need), None)
    assert st == 1 and not h.value and b"2^32" in lib.tnmc_last_error(None)


def test_closed_form_bond_dimensions_match_recurrences():
    """tnmc_common.cuh row_bond() / model.row_bond(): min(chi, 2^min(c, L-c), 2^(L-r)) equals the
    recurrences q_{c+1} = min(2 q_c, D'_{c+1}), k_c = min(chi, q_c, 2 k_{c+1}) of reading P-C2."""
    from paper_2509_19006_b200.model import row_bond
    for L in range(2, 18):
        for chi in (2, 3, 4, 5, 7, 8, 12, 16, 32):
            b = [1] + [2] * (L - 1) + [1]
            for r in range(L - 2, -1, -1):
                dp = [1] + [2 * b[c] for c in range(1, L)] + [1]
                q = [1] * (L + 1)
                for c in range(L - 1):
                    q[c + 1] = min(2 * q[c], dp[c + 1])
                k = [1] * (L + 1)
                for c in range(L - 1, 0, -1):
                    k[c] = min(chi, q[c], 2 * k[c + 1])
                b = k
                assert b == [row_bond(L, chi, r, c) for c in range(L + 1)]


def test_bond_dimensions_match_the_oracle_shapes():
    from oracle import bmps
    from paper_2509_19006_b200.model import row_bond
    from tnmc_workloads import make_couplings
    L, chi = 9, 5
    Jr, Jd = make_couplings(L, 1, 3)
    cache, _ = bmps.build_cache(Jr[0], Jd[0], 0.8, chi)
    for r in range(L):
        for c in range(L):
            assert cache[r][c].shape == (row_bond(L, chi, r, c), 2, row_bond(L, chi, r, c + 1))


def test_work_model():
    from paper_2509_19006_b200 import model
    # bond-saturated rows cost ~181 chi^3 per site: QR 26.7 + Q 26.7 + R.C 8 + Q.Pc 16 + SVD 96 + M.V 8
    f = model.build_flops_per_disorder(256, 16)
    per = f / (255 * 256 * 16 ** 3)
    assert 165 < per < 182
    assert model.sample_flops_per_chain_site(32) == 8192
    assert model.pad_chi(2) == 8 and model.pad_chi(9) == 16 and model.pad_chi(17) == 32


def test_bitpack_roundtrip():
    from bitpack import pack, unpack
    rng = np.random.default_rng(0)
    for L in (2, 31, 32, 33, 70):
        cfg = rng.integers(0, 2, (2, 3, L, L))
        w = pack(cfg)
        assert w.shape == (2, 3, L, (L + 31) // 32) and w.dtype == np.uint32
        assert (unpack(w, L) == cfg).all()
        assert w[0, 0, 0, 0] & 1 == cfg[0, 0, 0, 0]


def test_slot_plan_of_the_checkpoint_policy():
    """Mirror of csrc/tnmc_ctx.cuh Plan: every row a segment samples is stored, rebuilt rows never
    overwrite the row they are built from."""
    def plan(L, k):
        n_seg = (L + k - 1) // k
        perm = lambda r: n_seg if r == L - 1 else (r // k if r % k == 0 else -1)
        seg_slot = lambda i: n_seg + 1 + i
        for j in range(n_seg):
            lo, hi = j * k, min((j + 1) * k, L)
            start = min((j + 1) * k, L - 1)
            slots = {}
            for r in range(lo, hi):
                slots[r] = perm(r) if perm(r) >= 0 else seg_slot(r - lo - 1)
            assert perm(start) >= 0
            used = list(slots.values()) + ([perm(start)] if start not in slots else [])
            assert len(set(used)) == len(used)
            assert max(used) < n_seg + 1 + max(k - 1, 2)
    for L in (2, 5, 8, 9, 12, 33):
        for k in range(1, L):
            plan(L, k)
