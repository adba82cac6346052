"""Seeded synthetic inputs shared by the oracle-side tests, the GPU tests and bench.py.

Holds none of the method's arithmetic: only the iid +-J coupling generator (the paper's
workload: each grid edge is -1 with probability p, +1 otherwise, open
boundaries; the Edwards-Anderson +-J model of the paper's results is p = 0.5,
PAPER.md:282-286) and the table of BASELINE.json configs.  The paper's numpy/networkx RNG
stream (`create_rbim`) is not reproduced: any iid +-J instance is an
equally valid workload (input recipe).
"""
import numpy as np

# BASELINE.json configs[i] -> (L, chi, betas, n_dis, n_samples, instance seed, sampling seed)
CONFIGS = {
    "C1": dict(L=8, chi=16, betas=(1.0,), n_dis=4, n_samples=64, inst_seed=1001, seed=2001),
    "C2": dict(L=32, chi=16, betas=(0.5, 1.0, 2.0), n_dis=100, n_samples=100, inst_seed=1002, seed=2002),
    "C3": dict(L=128, chi=32, betas=(1.0,), n_dis=256, n_samples=256, inst_seed=1003, seed=2003),
    "C4": dict(L=512, chi=32, betas=(1.0,), n_dis=500, n_samples=200, inst_seed=1004, seed=2004),
    "C5": dict(L=1024, chi=32, betas=(1.0,), n_dis=1000, n_samples=1000, inst_seed=1005, seed=2005),
    # profiling shape: C3's kernels, grid (256 CTAs, two per SM) and per-site work at a quarter of the rows and columns, so that
    # an `ncu --set full` capture (about 40 replays with device memory saved and restored around each) takes minutes
    "C3q": dict(L=64, chi=32, betas=(1.0,), n_dis=256, n_samples=256, inst_seed=1003, seed=2003),
    # context only: the paper's own headline setting (chi = 8), in FP64 here
    "C5p": dict(L=1024, chi=8, betas=(1.0,), n_dis=1000, n_samples=1000, inst_seed=1005, seed=2005),
}


def make_couplings(L, n_dis, inst_seed, p=0.5, first_disorder=0):
    """Jr, Jd: int8 (n_dis, L, L).  Jr[d,r,c] couples (r,c)-(r,c+1), 0 at c=L-1;
    Jd[d,r,c] couples (r,c)-(r+1,c), 0 at r=L-1.  Disorder d's instance depends only on
    (inst_seed, first_disorder + d, L), not on n_dis."""
    Jr = np.zeros((n_dis, L, L), dtype=np.int8)
    Jd = np.zeros((n_dis, L, L), dtype=np.int8)
    for d in range(n_dis):
        rng = np.random.default_rng([int(inst_seed), int(first_disorder + d), int(L)])
        Jr[d, :, : L - 1] = np.where(rng.random((L, L - 1)) < p, -1, 1)
        Jd[d, : L - 1, :] = np.where(rng.random((L - 1, L)) < p, -1, 1)
    return Jr, Jd


def make_gaussian_couplings(L, n_dis, inst_seed, first_disorder=0):
    """Gaussian Edwards-Anderson couplings J ~ N(0, 1) on every bond of the open L x L grid (SURVEY 8f
    NEXT-1); float64 (n_dis, L, L), zero on the open boundary.  Same indexing as make_couplings."""
    Jr = np.zeros((n_dis, L, L))
    Jd = np.zeros((n_dis, L, L))
    for d in range(n_dis):
        rng = np.random.default_rng([int(inst_seed), int(first_disorder + d), int(L), 7])
        Jr[d, :, : L - 1] = rng.standard_normal((L, L - 1))
        Jd[d, : L - 1, :] = rng.standard_normal((L - 1, L))
    return Jr, Jd


def to_paper_layout(Jr, Jd):
    """(..., L, L, 4) float32 tensor (left, up, right, down) of PAPER.md:127, zeros at open edges."""
    J = np.zeros(Jr.shape + (4,), dtype=np.float32)
    J[..., 2] = Jr
    J[..., 3] = Jd
    J[..., :, 1:, 0] = Jr[..., :, :-1]
    J[..., 1:, :, 1] = Jd[..., :-1, :]
    return J
