"""Oracle Part C: boundary-MPS cache build (test infrastructure, see oracle/__init__.py).

Follows `create_cache_ising` step by step for ONE disorder realisation;
the disorder axis of PAPER.md:270 is a plain loop in the callers.  numpy, FP64.

Index conventions of the listing: MPS tensor (left bond, physical, right bond)
(PAPER.md:145); MPO tensor (left, physical-up, right, down) (shapes at PAPER.md:145,
einsums at :176, :182).  Couplings: the paper's J_mat[r,c,2] (right) is Jr[r,c] here,
J_mat[r,c,3] (down) is Jd[r,c], J_mat[r,c,1] (up) is Jd[r-1,c].

`multiply` and `compress` are named but not shown in the paper.
`multiply` is the standard MPO x MPS contraction of Fig. 2.  `compress`
follows reading P-C2 of DESIGN.md ("parity unpinned" against the paper's own code):
  1. left->right:  thin QR of (D_l*2) x D_r, A_c <- Q, s = |R|_F, logscale += log s,
                   A_{c+1} <- (R/s) A_{c+1}
  2. right->left:  SVD of D_l x (2*D_r), keep the k = min(chi, D_l, 2*D_r) largest singular
                   values, no value threshold, A_c <- V_k^T, A_{c-1} <- A_{c-1} (M V_k)
  3. s = |A_0|_F, logscale += log s, A_0 /= s.
The stored row state Psihat_r has unit 2-norm as a 2^L vector; Psi_r = exp(logscale_r) Psihat_r.
numpy.linalg.qr / numpy.linalg.svd (LAPACK) serve as library steps.
"""
import numpy as np


def set_ising_bmat(beta, J):
    """Eq. 7: rows/cols are s in {-1,+1}."""
    s = np.array([-1.0, 1.0])
    return np.exp(beta * float(J) * np.outer(s, s))


def copy_tensors():
    """Eq. 8 and PAPER.md:155-156 ('12' is a garbled I2)."""
    I2 = np.eye(2)
    I3 = np.zeros((2, 2, 2))
    I4 = np.zeros((2, 2, 2, 2))
    for i in range(2):
        I3[i, i, i] = 1.0
        I4[i, i, i, i] = 1.0
    return I2, I3, I4


def bottom_mps(Jr, beta):
    """C0: MPS of row L-1, shapes [(1,2,2),(2,2,2)...,(2,2,1)]."""
    L = Jr.shape[0]
    I2, I3, _ = copy_tensors()
    mps = [(I2 @ set_ising_bmat(beta, Jr[L - 1, 0]))[None, :, :]]
    for col in range(1, L - 1):
        mps.append(I3 @ set_ising_bmat(beta, Jr[L - 1, col]))
    mps.append(I2[:, :, None])
    return mps


def row_mpo(Jr, Jd, beta, row):
    """C1: MPO of one row, shapes [(1,2,2,2),(2,2,2,2)...,(2,2,1,2)].
    The interior append line is missing from the listing (:177-180); reading G4:
    W[l,a,r,d] = sum_xy I4[l,a,x,y] B_r[x,r] B_d[y,d]."""
    L = Jr.shape[0]
    _, I3, I4 = copy_tensors()
    mpo = []
    B_d = set_ising_bmat(beta, Jd[row, 0]); B_r = set_ising_bmat(beta, Jr[row, 0])
    mpo.append(np.einsum("ijk,jl,km->ilm", I3, B_r, B_d)[None])
    for col in range(1, L - 1):
        B_d = set_ising_bmat(beta, Jd[row, col]); B_r = set_ising_bmat(beta, Jr[row, col])
        mpo.append(np.einsum("laxy,xr,yd->lard", I4, B_r, B_d))
    B_d = set_ising_bmat(beta, Jd[row, L - 1])
    mpo.append(np.einsum("ijk,kl->ijl", I3, B_d)[:, :, None, :])
    return mpo


def multiply(mpo, mps):
    """Fig. 2: A'[(l,i),a,(r,k)] = sum_m W[l,a,r,m] A[i,m,k]; bonds multiply."""
    out = []
    for W, A in zip(mpo, mps):
        T = np.einsum("larm,imk->liark", W, A)
        l, i, a, r, k = T.shape
        out.append(T.reshape(l * i, a, r * k))
    return out


def compress(mps, chi):
    """Reading P-C2 (module docstring). Returns (logscale, mps, discarded) where
    discarded[c] = sum of squared singular values dropped at the bond left of site c,
    divided by the squared norm of the (canonicalised) state before any truncation."""
    mps = [A.copy() for A in mps]
    L = len(mps)
    logscale = 0.0
    for c in range(L - 1):                                   # 1. left -> right QR
        Dl, d, Dr = mps[c].shape
        Q, R = np.linalg.qr(mps[c].reshape(Dl * d, Dr))
        s = np.linalg.norm(R)
        logscale += np.log(s)
        mps[c] = Q.reshape(Dl, d, Q.shape[1])
        mps[c + 1] = np.einsum("xi,iak->xak", R / s, mps[c + 1])
    discarded = np.zeros(L)
    norm2 = float(np.linalg.norm(mps[L - 1]) ** 2)           # sites 0..L-2 are isometries now
    for c in range(L - 1, 0, -1):                            # 2. right -> left truncated SVD
        Dl, d, Dr = mps[c].shape
        M = mps[c].reshape(Dl, d * Dr)
        _, S, Vt = np.linalg.svd(M, full_matrices=False)
        k = min(chi, Dl, d * Dr)
        discarded[c] = float((S[k:] ** 2).sum()) / norm2
        Vk = Vt[:k].T                                        # (d*Dr, k)
        mps[c] = Vt[:k].reshape(k, d, Dr)
        mps[c - 1] = np.einsum("iak,kx->iax", mps[c - 1], M @ Vk)
    s = np.linalg.norm(mps[0])                               # 3. final scale
    logscale += np.log(s)
    mps[0] = mps[0] / s
    return logscale, mps, discarded


def build_cache(Jr, Jd, beta, chi):
    """C0-C2 for one disorder: returns (cache, logscale) with cache[r] = MPS of rows r..L-1
    (list of L tensors) and logscale[r] such that
    Psi_r = exp(logscale[r]) * Psihat_r.  Row L-1 is stored as built."""
    L = Jr.shape[0]
    cache = [None] * L
    logscale = np.zeros(L)
    mps = bottom_mps(Jr, beta)
    cache[L - 1] = mps
    for row in range(L - 2, -1, -1):
        mpo = row_mpo(Jr, Jd, beta, row)
        mps = multiply(mpo, mps)
        ls, mps, _ = compress(mps, chi)
        cache[row] = mps
        logscale[row] = logscale[row + 1] + ls
    return cache, logscale


def log_z(mps_row0, logscale0):
    """C3: log Z = logscale_0 + log |sum_sigma Psihat_0(sigma)| (Eq. 6), the sum
    taken as the product over c of sum_a A_c[:,a,:] with a running rescale.  Returns
    (logZ, sign) so that a non-positive sum can be flagged."""
    v = np.ones(1)
    lg = float(logscale0)
    for A in mps_row0:
        v = v @ A.sum(axis=1)
        m = np.abs(v).max()
        if m == 0.0:
            return -np.inf, 0.0
        v = v / m
        lg += np.log(m)
    return lg + np.log(abs(v[0])), float(np.sign(v[0]))


def mps_to_vector(mps):
    """Expand an MPS to its 2^L vector; bit c of the index is a_c. Small L only (pins)."""
    L = len(mps)
    t = mps[0][0]                                            # (a0, D)
    for A in mps[1:]:
        t = np.tensordot(t, A, axes=([-1], [0]))             # (a0..ac, D)
    t = t[..., 0]                                            # (a0, a1, ..., a_{L-1})
    return np.transpose(t, list(range(L - 1, -1, -1))).reshape(-1)
