"""Algorithmic work of the hot path ("Roofline"): nominal flops of the boundary-MPS build
per disorder and flops / bytes of the sampler per chain-site.  Pure counting -- no arithmetic of the
method lives here.  The counts use the actual bond dimensions of every site (edges of the lattice
and the first rows are not saturated at chi)."""


def row_bond(L, chi, r, c):
    """Bond dimension left of column c of stored row r: min(chi, 2^min(c, L-c), 2^(L-r)); 1 at the ends."""
    if c <= 0 or c >= L:
        return 1
    e = min(c, L - c, L - r)
    return chi if e >= 6 else min(chi, 1 << e)


def _qr_flops(m, n):
    """Householder QR of an m x n matrix, R only (Golub & Van Loan): 2 n^2 (m - n/3) for m >= n."""
    if m < n:
        m, n = n, m
    return 2.0 * n * n * (m - n / 3.0)


def build_flops_per_disorder(L, chi):
    """Nominal FP64 flops of tnmc_build_envs for one disorder (QR + form-Q + R.C +
    SVD(Sigma, V) + M.V + Q.(MV); 205 chi^3 per bond-saturated site-row)."""
    total = 0.0
    for r in range(L - 2, -1, -1):
        q = [1] * (L + 1)
        for c in range(L - 1):
            d_next = 2 * row_bond(L, chi, r + 1, c + 1)
            q[c + 1] = min(2 * q[c], d_next)
        q[L] = 1
        k_next = 1
        for c in range(L - 1, -1, -1):
            bl, br = row_bond(L, chi, r + 1, c), row_bond(L, chi, r + 1, c + 1)
            m = 2 * q[c]
            n = (1 if c == L - 1 else 2) * br
            total += 2.0 * 2 * q[c] * bl * br              # T_a = R_a C_a, both spin slices
            if c < L - 1:
                total += 2.0 * _qr_flops(m, n)             # QR and the explicit Q
            total += 2.0 * m * q[c + 1] * k_next           # M = Q_c Pc
            if c > 0:
                nr, nc = q[c], 2 * k_next
                total += 12.0 * nr * nc * min(nr, nc)      # SVD, singular values and one set of vectors
                k = min(chi, nr, nc)
                total += 2.0 * nr * nc * k                 # M V_k
                k_next = k
    return total


def sample_flops_per_chain_site(P):
    """8 P^2: two (1 x P) x (P x 2P) products per site (right and left sweep), P = padded chi."""
    return 8.0 * P * P


def sample_bytes_per_chain_site(P, n_chains_per_tile=128, w=8):
    """HBM bytes per chain-site: the right environment written once and read once (2 P w), one
    spin bit, and the site tensor (2 P^2 w) read twice per row by every CTA of n_chains_per_tile chains."""
    return 2.0 * P * w + 0.125 + 2.0 * (2 * P * P * w) / n_chains_per_tile


def pad_chi(chi):
    return 8 if chi <= 8 else (16 if chi <= 16 else 32)
