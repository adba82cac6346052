// tnmc_build.cuh -- boundary-MPS environment build (steps a-1..a-7 of DESIGN.md).
//
// One CTA per disorder realisation walks the rows bottom -> top and, per row,
//   1. applies the row MPO (Eq. 7-8) site by site, fused with
//   2. the left->right canonicalising Householder QR sweep (P-C2 step 1), then
//   3. the right->left truncated SVD sweep (P-C2 step 2; one-sided Jacobi on the rows of the
//      D_l x 2D_r matrix) and the final scale (P-C2 step 3).
// The MPO tensors are never materialised: with W[l,a,r,d] = delta(l,a) B_r[a,r] B_d[a,d]
// the product tensor is  A'[(l,i),a,(r,k)] = delta(l,a) B_r[a,r] C_a[i,k],
// C_a = sum_m B_d[a,m] A[i,m,k], so the carried R of the QR sweep only ever meets C_a.
#pragma once
#include "tnmc_common.cuh"
#include "tnmc_linalg.cuh"

namespace tnmc {

constexpr int BUILD_THREADS = 256;

#ifdef TNMC_PROFILE
#define PROF_DECL long long prof_t0 = clock64();
#define PROF(slot) do { if (blockIdx.x == 0 && threadIdx.x == 0) { const long long t_ = clock64(); atomicAdd(&g_build_prof[slot], (unsigned long long)(t_ - prof_t0)); prof_t0 = t_; } } while (0)
#define PROF_ADD(slot, v) do { if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(&g_build_prof[slot], (unsigned long long)(v)); } while (0)
#else
#define PROF_DECL
#define PROF(slot)
#define PROF_ADD(slot, v)
#endif

struct BuildArgs {
    JView J;
    double beta;
    int L, chi;
    int dis_begin;               // CTA b works on disorder dis_begin + b
    int row_hi, row_lo;          // processes rows row_hi-1, ..., row_lo; row row_hi must be stored
    const int* slot_of_row;      // [L] device: env slot of each row for this pass (-1: not stored)
    double* env;                 // env base
    size_t env_dis_stride;       // doubles per disorder (n_slots * L * 2P^2)
    double* qbuf;                // scratch, per disorder L * (LDX * D) doubles
    double* logscale;            // (n_dis, L): logscale of every row (written for rows built)
    unsigned long long* flags;
};

template <int P>
struct BuildCfg {
    static constexpr int D = 2 * P;           // doubled bond
    static constexpr int LDX = 2 * D + 1;     // leading dim of the column-major QR operand (odd: no bank conflicts)
    static constexpr int LDM = 2 * P;         // row length of the Jacobi operand (row-major)
    static constexpr int LDV = 2 * P + 1;     // padded row length of the selected right singular vectors
    static constexpr int TSZ = 2 * P * P;     // doubles per stored site tensor
    static constexpr int QSZ = LDX * D;       // doubles per site of the Q scratch
    // shared-memory carve-up (doubles)
    static constexpr int X_OFF = 0;                   // LDX*D : QR operand / Q_c / staging
    static constexpr int R_OFF = X_OFF + LDX * D;     // D*LDC : carried R [x][lambda] (ld D) / column-major M for QRCP (ld LDC)
    static constexpr int LDC = D + 1;         // leading dim of the column-major copy of M that QRCP works on
    static constexpr int A_OFF = R_OFF + D * LDC;     // TSZ   : lower-row site tensor (fragment order) / Pc
    static constexpr int C_OFF = A_OFF + TSZ;         // TSZ   : C_a[i][k] / Pc_new
    static constexpr int M0_OFF = C_OFF + TSZ;        // D*LDM : copy of M before rotation
    static constexpr int S_OFF = M0_OFF + D * LDM;    // 2*D + 8 : tau / sigma / scalars
    static constexpr int N_DBL = S_OFF + 2 * D + 8;
    static size_t smem_bytes(int L) { return sizeof(double) * N_DBL + sizeof(int) * (L + 2 + 2 * D); }
};

template <int P>
__global__ void __launch_bounds__(BUILD_THREADS, 1) build_rows_kernel(const BuildArgs args) {
    using Cfg = BuildCfg<P>;
    constexpr int D = Cfg::D, LDX = Cfg::LDX, LDM = Cfg::LDM, LDV = Cfg::LDV, TSZ = Cfg::TSZ, LDC = Cfg::LDC;
    extern __shared__ __align__(16) double smem[];
    double* sX = smem + Cfg::X_OFF;
    double* sR = smem + Cfg::R_OFF;
    double* sA = smem + Cfg::A_OFF;
    double* sC = smem + Cfg::C_OFF;
    double* sM0 = smem + Cfg::M0_OFF;
    double* sS = smem + Cfg::S_OFF;      // [0,D): tau / sigma   [D, 2D): reduction scratch
    double* sRed = sS + D;
    int* sq = reinterpret_cast<int*>(smem + Cfg::N_DBL);   // [L+1] QR bond dims
    int* spos = sq + args.L + 2;                           // [2D] rank / position of each Jacobi row

    const int tid = threadIdx.x;
    const int d = args.dis_begin + blockIdx.x;
    const int L = args.L, chi = args.chi;
    const double beta = args.beta;
    double* env_d = args.env + (size_t)d * args.env_dis_stride;
    double* qbuf_d = args.qbuf + (size_t)d * (size_t)L * Cfg::QSZ;
    double* ls_d = args.logscale + (size_t)d * L;

    PROF_DECL
    for (int r = args.row_hi - 1; r >= args.row_lo; --r) {
        const double* env_in = env_d + (size_t)args.slot_of_row[r + 1] * L * TSZ;
        double* env_out = env_d + (size_t)args.slot_of_row[r] * L * TSZ;
        double logs = 0.0;   // all threads carry the same value

        // ------------------------------------------------------------------ QR sweep, left -> right
        if (tid == 0) { sq[0] = 1; sR[0] = 1.0; sR[1] = 1.0; }
        __syncthreads();
        for (int c = 0; c < L; ++c) {
            const int bl = row_bond(L, chi, r + 1, c), br = row_bond(L, chi, r + 1, c + 1);
            const int ql = sq[c], m = 2 * ql;
            const int nr = (c == L - 1) ? 1 : 2, n = nr * br;
            const double* Ain = env_in + (size_t)c * TSZ;
            for (int t = tid; t < TSZ; t += BUILD_THREADS) sA[t] = Ain[t];
            __syncthreads();
            {   // C_a[i][k] = sum_m B_d[a][m] A[i][m][k]      (Eq. 7: B_d[a][m] = exp(beta Jd (2a-1)(2m-1)))
                const int jd = args.J.jd(d, r, c);
                const double w_same = exp(beta * jd), w_diff = exp(-beta * jd);
                for (int t = tid; t < 2 * bl * br; t += BUILD_THREADS) {
                    const int k = t % br, i = (t / br) % bl, a = t / (br * bl);
                    sC[(a * P + i) * P + k] = w_same * sA[env_off(P, i, a, k)] + w_diff * sA[env_off(P, i, 1 - a, k)];
                }
            }
            __syncthreads();
            {   // X[(2x+a), (rr*br+k)] = B_r[a][rr] * sum_i R[x][a*bl+i] C_a[i][k]
                const int jr = (c == L - 1) ? 0 : args.J.jr(d, r, c);
                const double w_same = exp(beta * jr), w_diff = exp(-beta * jr);
                for (int t = tid; t < m * br; t += BUILD_THREADS) {
                    const int k = t % br, a = (t / br) & 1, x = t / (2 * br);
                    const double* Rrow = sR + (size_t)x * D + a * bl;
                    const double* Ccol = sC + (size_t)a * P * P + k;
                    double acc = 0.0;
                    for (int i = 0; i < bl; ++i) acc += Rrow[i] * Ccol[i * P];
                    const int row = 2 * x + a;
                    if (nr == 1) sX[row + (size_t)k * LDX] = acc;
                    else {
                        sX[row + (size_t)((a)*br + k) * LDX] = w_same * acc;       // rr == a
                        sX[row + (size_t)((1 - a) * br + k) * LDX] = w_diff * acc; // rr != a
                    }
                }
            }
            __syncthreads();
            double* Qout = qbuf_d + (size_t)c * Cfg::QSZ;
            if (c == L - 1) {
                // last site: not orthogonalised (P-C2 step 1 stops at L-2); it now carries the norm
                for (int t = tid; t < m; t += BUILD_THREADS) Qout[t] = sX[t];
                if (tid == 0) sq[L] = 1;
                __syncthreads();
                break;
            }
            PROF(0);
            householder_qr<P>(sX, LDX, m, n, sS);
            PROF(1);
            const int kk = m < n ? m : n;
            // R -> carried R/|R|_F for the next site; logscale += log |R|_F
            double ss = 0.0;
            for (int t = tid; t < kk * n; t += BUILD_THREADS) {
                const int x = t / n, lam = t % n;
                const double v = lam >= x ? sX[x + (size_t)lam * LDX] : 0.0;
                ss += v * v;
            }
            ss = block_sum(ss, sRed);
            const double s = sqrt(ss);
            if (!(s > 0.0) || !isfinite(s)) { if (tid == 0) raise_flag(args.flags, FLAG_NONFINITE); }
            logs += log(s);
            const double inv_s = 1.0 / s;
            for (int t = tid; t < kk * n; t += BUILD_THREADS) {
                const int x = t / n, lam = t % n;
                sR[(size_t)x * D + lam] = lam >= x ? sX[x + (size_t)lam * LDX] * inv_s : 0.0;
            }
            if (tid == 0) sq[c + 1] = kk;
            __syncthreads();
            PROF(2);
            householder_form_q<P>(sX, LDX, m, kk, sS);
            PROF(3);
            for (int t = tid; t < m * kk; t += BUILD_THREADS) {
                const int row = t % m, col = t / m;
                Qout[row + (size_t)col * LDX] = sX[row + (size_t)col * LDX];
            }
            __syncthreads();
        }

        // ------------------------------------------------------------------ SVD sweep, right -> left
        double* sMc = sR;         // M, column-major [x + col*LDC]: QRCP operand
        double* sM = sX;          // Jacobi operand (rows of R), row-major, ld = LDM; lives in sX once Q_c is consumed
        int* sperm = spos + D;    // column permutation of the QRCP
        double* sPc = sA;         // carried M V_k of the site to the right: [z][y], ld = P
        double* sPn = sC;
        int kprev = 1;
        if (tid == 0) sPc[0] = 1.0;
        __syncthreads();
        for (int c = L - 1; c >= 0; --c) {
            const int ql = sq[c], m = 2 * ql, qr = sq[c + 1];
            const double* Qin = qbuf_d + (size_t)c * Cfg::QSZ;
            for (int t = tid; t < m * qr; t += BUILD_THREADS) {
                const int row = t % m, col = t / m;
                sX[row + (size_t)col * LDX] = Qin[row + (size_t)col * LDX];
            }
            __syncthreads();
            const int nc = 2 * kprev;
            // M[x][a*kprev+y] = sum_z Q_c[(2x+a)][z] Pc[z][y]
            for (int t = tid; t < ql * nc; t += BUILD_THREADS) {
                const int y = t % kprev, a = (t / kprev) & 1, x = t / nc;
                const double* Xrow = sX + (2 * x + a);
                double acc = 0.0;
                for (int z = 0; z < qr; ++z) acc += Xrow[(size_t)z * LDX] * sPc[z * P + y];
                sMc[x + (size_t)(a * kprev + y) * LDC] = acc;
                sM0[(size_t)x * LDM + a * kprev + y] = acc;
            }
            __syncthreads();
            double* stage = sX + D * LDM;       // TSZ doubles: output tensor in fragment order
            double* sV = stage + TSZ;           // [y'][col], ld = LDV: selected right singular vectors
            for (int t = tid; t < TSZ; t += BUILD_THREADS) stage[t] = 0.0;
            double* Aout = env_out + (size_t)c * TSZ;
            if (c == 0) {
                // P-C2 step 3: A_0 (1,2,k_1) = Q_0 Pc; divide by its norm, add log to logscale
                double ss = 0.0;
                for (int t = tid; t < nc; t += BUILD_THREADS) ss += sM0[t] * sM0[t];
                ss = block_sum(ss, sRed);
                const double s = sqrt(ss);
                if (!(s > 0.0) || !isfinite(s)) { if (tid == 0) raise_flag(args.flags, FLAG_NONFINITE); }
                logs += log(s);
                const double inv_s = 1.0 / s;
                for (int t = tid; t < nc; t += BUILD_THREADS) {
                    const int y = t % kprev, a = t / kprev;
                    stage[env_off(P, 0, a, y)] = sM0[t] * inv_s;
                }
                __syncthreads();
                for (int t = tid; t < TSZ; t += BUILD_THREADS) Aout[t] = stage[t];
                __syncthreads();
                break;
            }
            // M P = Q R with column pivoting (R only); the singular values and right singular vectors of
            // M are those of R, with the columns permuted back
            PROF(7);
            const double fro2 = householder_qrcp<P / 2>(sMc, LDC, ql, nc, sRed, sperm, sS, nullptr);
            const int nrow = ql < nc ? ql : nc;        // rows of R (even: ql and nc are)
            for (int t = tid; t < nrow * nc; t += BUILD_THREADS) {
                const int j = t % nc, i = t / nc;
                sM[(size_t)i * LDM + j] = j >= i ? sMc[i + (size_t)j * LDC] : 0.0;
            }
            __syncthreads();
            const double thr2 = fro2 * 1e-30;      // sigma <= 1e-15 |M|_F: below the numerical rank
            PROF(4);
            const int nsw = jacobi_rows(sM, LDM, nrow, nc, fro2, thr2, sS, args.flags);
            PROF(5);
            PROF_ADD(8, nsw); PROF_ADD(9, 1);
            // singular values = row norms
            {
                const int grp = tid >> 3, t8 = tid & 7;
                for (int x = grp; x < nrow; x += (BUILD_THREADS >> 3)) {
                    double a = 0.0;
                    for (int cc = t8; cc < nc; cc += 8) { const double v = sM[(size_t)x * LDM + cc]; a += v * v; }
#pragma unroll
                    for (int o = 4; o > 0; o >>= 1) a += __shfl_xor_sync(0xffu << ((tid & 31) & ~7), a, o);
                    if (t8 == 0) sS[x] = sqrt(a);
                }
            }
            __syncthreads();
            int k = chi < ql ? chi : ql;
            if (nc < k) k = nc;
            for (int x = tid; x < nrow; x += BUILD_THREADS) {
                const double sx = sS[x];
                int rank = 0;
                for (int y = 0; y < nrow; ++y) {
                    const double sy = sS[y];
                    rank += (sy > sx) || (sy == sx && y < x);
                }
                spos[x] = rank < k ? rank : -1;
                if (rank < k && !(sx * sx > thr2)) raise_flag(args.flags, FLAG_SIGMA_ZERO);
            }
            __syncthreads();
            // A_c[y'][a][y] = v_{y'}  (rows of V_k^T), staged in fragment order and as plain rows
            for (int t = tid; t < nrow * nc; t += BUILD_THREADS) {
                const int col = t % nc, x = t / nc;
                const int yp = spos[x];
                if (yp >= 0) {
                    const double sx = sS[x];
                    // a kept direction below the numerical rank carries no weight (M v = 0 for any
                    // orthonormal completion); it is stored as a zero row
                    const double v = sx * sx > thr2 ? sM[(size_t)x * LDM + col] / sx : 0.0;
                    const int oc = sperm[col];        // original column (a, y) of pivoted column col
                    sV[(size_t)yp * LDV + oc] = v;
                    stage[env_off(P, yp, oc / kprev, oc % kprev)] = v;
                }
            }
            __syncthreads();
            for (int t = tid; t < TSZ; t += BUILD_THREADS) Aout[t] = stage[t];
            // Pn[x][y'] = sum_col M0[x][col] V_k[col][y']   (= M V_k, projector form of P-C2 step 2)
            for (int t = tid; t < ql * k; t += BUILD_THREADS) {
                const int yp = t % k, x = t / k;
                const double* mrow = sM0 + (size_t)x * LDM;
                const double* vrow = sV + (size_t)yp * LDV;
                double acc = 0.0;
                for (int col = 0; col < nc; ++col) acc += mrow[col] * vrow[col];
                sPn[x * P + yp] = acc;
            }
            __syncthreads();
            { double* t = sPc; sPc = sPn; sPn = t; }
            kprev = k;
            PROF(6);
        }
        if (tid == 0) ls_d[r] = ls_d[r + 1] + logs;
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Bottom-row MPS, written unnormalised exactly as the listing builds it:
//   A_0[0][a][b] = B(Jr[L-1][0])[a][b];  A_c[l][a][b] = delta(l,a) B(Jr[L-1][c])[a][b];
//   A_{L-1}[l][a][0] = delta(l,a).   One CTA per (site, disorder).
// ---------------------------------------------------------------------------------------------
__global__ void bottom_row_kernel(JView J, double beta, int L, int P, double* env, size_t env_dis_stride,
                                  int slot, double* logscale) {
    const int c = blockIdx.x, d = blockIdx.y;
    const int TSZ = 2 * P * P;
    double* A = env + (size_t)d * env_dis_stride + ((size_t)slot * L + c) * TSZ;
    for (int t = threadIdx.x; t < TSZ; t += blockDim.x) A[t] = 0.0;
    __syncthreads();
    if (threadIdx.x < 8) {
        const int l = threadIdx.x >> 2, a = (threadIdx.x >> 1) & 1, b = threadIdx.x & 1;
        const int jr = (c == L - 1) ? 0 : J.jr(d, L - 1, c);
        const double bm = exp(beta * jr * (2 * a - 1) * (2 * b - 1));
        if (c == 0) { if (l == 0) A[env_off(P, 0, a, b)] = bm; }
        else if (c == L - 1) { if (b == 0 && l == a) A[env_off(P, l, a, 0)] = 1.0; }
        else if (l == a) A[env_off(P, l, a, b)] = bm;
    }
    if (c == 0 && threadIdx.x == 0) logscale[(size_t)d * L + (L - 1)] = 0.0;
}

// ---------------------------------------------------------------------------------------------
// log Z read-out (a-7; Eq. 6): log Z = logscale_0 + log |sum_sigma Psihat_0(sigma)|,
// the sum taken as the product over c of sum_a A_c[:,a,:] with a running max-abs rescale.
// One warp per disorder; lane j carries component j of the running row vector.
// ---------------------------------------------------------------------------------------------
__global__ void logz_kernel(int L, int chi, int P, int n_dis, const double* env, size_t env_dis_stride,
                            int slot0, const double* logscale, double* logZ, unsigned long long* flags) {
    const int d = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (d >= n_dis) return;
    const int lane = threadIdx.x & 31;
    const int TSZ = 2 * P * P;
    const double* row = env + (size_t)d * env_dis_stride + (size_t)slot0 * L * TSZ;
    double v = lane == 0 ? 1.0 : 0.0;   // component `lane` of the running vector (P <= 32)
    double lg = logscale[(size_t)d * L];
    for (int c = 0; c < L; ++c) {
        const double* A = row + (size_t)c * TSZ;
        const int bl = row_bond(L, chi, 0, c), br = row_bond(L, chi, 0, c + 1);
        double acc = 0.0;
        for (int i = 0; i < bl; ++i) {
            const double vi = __shfl_sync(0xffffffffu, v, i);
            if (lane < br) acc += vi * (A[env_off(P, i, 0, lane)] + A[env_off(P, i, 1, lane)]);
        }
        double mx = fabs(acc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if (!(mx > 0.0)) { if (lane == 0) { logZ[d] = -INFINITY; raise_flag(flags, FLAG_LOGZ_NONPOS); } return; }
        v = acc / mx;
        lg += log(mx);
    }
    const double v0 = __shfl_sync(0xffffffffu, v, 0);
    if (lane == 0) {
        if (!(v0 > 0.0)) raise_flag(flags, FLAG_LOGZ_NONPOS);
        logZ[d] = lg + log(fabs(v0));
    }
}

// ---------------------------------------------------------------------------------------------
// Pack int8 couplings into bit masks (see tnmc_common.cuh).  One thread per (mask word).
// ---------------------------------------------------------------------------------------------
__global__ void pack_couplings_kernel(const int8_t* Jr, const int8_t* Jd, int n_dis, int L, int W,
                                      uint32_t* masks) {
    const size_t n_words = (size_t)n_dis * L * W;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_words) return;
    const int w = idx % W;
    const size_t dr = idx / W;   // d*L + r
    uint32_t rn = 0, rz = 0, dn = 0, dz = 0;
    for (int b = 0; b < 32; ++b) {
        const int c = w * 32 + b;
        if (c >= L) break;
        const int8_t jr = Jr[dr * L + c], jd = Jd[dr * L + c];
        rn |= (uint32_t)(jr < 0) << b; rz |= (uint32_t)(jr != 0) << b;
        dn |= (uint32_t)(jd < 0) << b; dz |= (uint32_t)(jd != 0) << b;
    }
    masks[0 * n_words + idx] = rn;
    masks[1 * n_words + idx] = rz;
    masks[2 * n_words + idx] = dn;
    masks[3 * n_words + idx] = dz;
}

// Export one stored row in the paper's layout (L, chi, 2, chi) -- test/inspection hook.
__global__ void export_row_kernel(int L, int chi, int P, const double* row, double* out) {
    const int c = blockIdx.x;
    const int TSZ = 2 * P * P;
    for (int t = threadIdx.x; t < chi * 2 * chi; t += blockDim.x) {
        const int j = t % chi, a = (t / chi) & 1, i = t / (2 * chi);
        out[(size_t)c * chi * 2 * chi + t] = row[(size_t)c * TSZ + env_off(P, i, a, j)];
    }
}

}  // namespace tnmc
