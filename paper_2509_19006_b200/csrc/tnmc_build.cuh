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

namespace tnmc {

constexpr int BUILD_THREADS = 256;

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
    static constexpr int R_OFF = X_OFF + LDX * D;     // D*D   : carried R [x][lambda] / Jacobi operand M
    static constexpr int A_OFF = R_OFF + D * D;       // TSZ   : lower-row site tensor (fragment order) / Pc
    static constexpr int C_OFF = A_OFF + TSZ;         // TSZ   : C_a[i][k] / Pc_new
    static constexpr int M0_OFF = C_OFF + TSZ;        // D*LDM : copy of M before rotation
    static constexpr int S_OFF = M0_OFF + D * LDM;    // 2*D + 8 : tau / sigma / scalars
    static constexpr int N_DBL = S_OFF + 2 * D + 8;
    static size_t smem_bytes(int L) { return sizeof(double) * N_DBL + sizeof(int) * (L + 2 + 2 * D); }
};

// block-wide sum of one double per thread; result valid in all threads. scratch: >= 32 doubles
__device__ __forceinline__ double block_sum(double v, double* scratch) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) scratch[w] = v;
    __syncthreads();
    double t = 0.0;
    const int nw = blockDim.x >> 5;
    for (int i = 0; i < nw; ++i) t += scratch[i];
    return t;
}

// Householder QR of the m x n column-major matrix X (leading dim ld) in shared memory.
// On return the upper trapezoid holds R, the reflector vectors (v_j, unit diagonal implied) sit
// below the diagonal, tau[j] their scalars; kk = min(m,n) reflectors.
__device__ void householder_qr(double* X, int ld, int m, int n, double* tau) {
    const int kk = m < n ? m : n;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    for (int j = 0; j < kk; ++j) {
        double* colj = X + (size_t)j * ld;
        if (warp == 0) {
            double ss = 0.0;
            for (int i = j + 1 + lane; i < m; i += 32) { const double v = colj[i]; ss += v * v; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
            const double alpha = colj[j];
            double t = 0.0, scale = 0.0, bet = alpha;
            if (ss != 0.0) {
                const double nrm = sqrt(alpha * alpha + ss);
                bet = alpha >= 0.0 ? -nrm : nrm;
                t = (bet - alpha) / bet;
                scale = 1.0 / (alpha - bet);
            }
            __syncwarp();
            for (int i = j + 1 + lane; i < m; i += 32) colj[i] *= scale;
            if (lane == 0) { colj[j] = bet; tau[j] = t; }
        }
        __syncthreads();
        const double t = tau[j];
        if (t != 0.0) {
            for (int jj = j + 1 + warp; jj < n; jj += nwarps) {
                double* col = X + (size_t)jj * ld;
                double w = 0.0;
                for (int i = j + 1 + lane; i < m; i += 32) w += colj[i] * col[i];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
                w += col[j];
                w *= t;
                __syncwarp();
                for (int i = j + 1 + lane; i < m; i += 32) col[i] -= w * colj[i];
                if (lane == 0) col[j] -= w;
            }
        }
        __syncthreads();
    }
}

// Overwrite the reflectors with the explicit thin Q (m x kk), in place (LAPACK dorg2r order).
__device__ void householder_form_q(double* X, int ld, int m, int kk, const double* tau) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    for (int j = kk - 1; j >= 0; --j) {
        double* colj = X + (size_t)j * ld;
        const double t = tau[j];
        if (t != 0.0) {
            for (int jj = j + 1 + warp; jj < kk; jj += nwarps) {
                double* col = X + (size_t)jj * ld;
                double w = 0.0;
                for (int i = j + 1 + lane; i < m; i += 32) w += colj[i] * col[i];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
                // row j of the trailing block is e_j-free here: Q[j][jj] = 0 before H_j is applied
                w *= t;
                __syncwarp();
                for (int i = j + 1 + lane; i < m; i += 32) col[i] -= w * colj[i];
                if (lane == 0) col[j] = -w;
            }
        } else {
            for (int jj = j + 1 + warp; jj < kk; jj += nwarps)
                if (lane == 0) X[(size_t)jj * ld + j] = 0.0;
        }
        __syncthreads();
        for (int i = threadIdx.x; i < m; i += blockDim.x) {
            double v;
            if (i < j) v = 0.0;
            else if (i == j) v = 1.0 - t;
            else v = -t * colj[i];
            colj[i] = v;
        }
        __syncthreads();
    }
}

// One-sided (Hestenes) Jacobi on the ROWS of the n x nc row-major matrix M (row length ld):
// plane rotations from the left until all rows are mutually orthogonal, so that row x ends as
// sigma_x * v_x^T (M = U Sigma V^T).  n must be even (callers pad with a zero row).
// Eight threads cooperate on one row pair; pairs follow the round-robin (circle) schedule.
// Returns the number of sweeps done (all threads).
// Rows whose squared norm is <= thr2 (numerically zero against |M|_F) are left alone: when M has
// more rows than its rank they only carry rounding noise, and chasing their orthogonality would
// grind them down to denormals without ever meeting the relative criterion.
__device__ int jacobi_rows(double* M, int ld, int n, int nc, double thr2, unsigned long long* flags) {
    const int grp = threadIdx.x >> 3, t8 = threadIdx.x & 7;
    const int npairs = n >> 1;
    const unsigned gmask = 0xffu << ((threadIdx.x & 31) & ~7);
    // A pair is rotated whenever its cosine exceeds one rounding error; the sweeps stop after the
    // first one in which every cosine met was below 1e-8: cyclic Jacobi converges quadratically, so
    // the rotations of that last sweep leave the rows orthogonal to rounding level (the accuracy
    // LAPACK's SVD gives the oracle).  A looser stop (cosines ~1e-14) was measurably not enough:
    // the row-to-row map amplifies such errors by up to ~1e6 ("Tolerances").
    const double rot2 = 4.930380657631324e-32;     // (2^-52)^2
    const double big2 = 1e-16;                     // (1e-8)^2
    int sweep = 0;
    for (; sweep < 60; ++sweep) {
        int any = 0;
        for (int round = 0; round < n - 1; ++round) {
            int rotated = 0;
            for (int p = grp; p < npairs; p += (blockDim.x >> 3)) {
                int r1, r2;
                if (p == 0) { r1 = n - 1; r2 = round; }
                else {
                    r1 = (round + p) % (n - 1);
                    r2 = (round - p + (n - 1)) % (n - 1);
                }
                if (r1 > r2) { const int t = r1; r1 = r2; r2 = t; }
                double* x = M + (size_t)r1 * ld;
                double* y = M + (size_t)r2 * ld;
                double a = 0.0, b = 0.0, g = 0.0;
                for (int c = 2 * t8; c < nc; c += 16) {
                    const double x0 = x[c], y0 = y[c];
                    a += x0 * x0; b += y0 * y0; g += x0 * y0;
                    if (c + 1 < nc) {
                        const double x1 = x[c + 1], y1 = y[c + 1];
                        a += x1 * x1; b += y1 * y1; g += x1 * y1;
                    }
                }
#pragma unroll
                for (int o = 4; o > 0; o >>= 1) {
                    a += __shfl_xor_sync(gmask, a, o);
                    b += __shfl_xor_sync(gmask, b, o);
                    g += __shfl_xor_sync(gmask, g, o);
                }
                if (a > thr2 && b > thr2 && g * g > rot2 * (a * b)) {
                    rotated |= g * g > big2 * (a * b);
                    const double zeta = (b - a) / (2.0 * g);
                    const double tt = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                    const double cs = 1.0 / sqrt(1.0 + tt * tt);
                    const double sn = cs * tt;
                    for (int c = 2 * t8; c < nc; c += 16) {
                        const double x0 = x[c], y0 = y[c];
                        x[c] = cs * x0 - sn * y0;
                        y[c] = sn * x0 + cs * y0;
                        if (c + 1 < nc) {
                            const double x1 = x[c + 1], y1 = y[c + 1];
                            x[c + 1] = cs * x1 - sn * y1;
                            y[c + 1] = sn * x1 + cs * y1;
                        }
                    }
                }
            }
            any |= __syncthreads_or(rotated);
        }
        if (!any) break;
    }
    if (sweep >= 60 && threadIdx.x == 0) raise_flag(flags, FLAG_JACOBI_LIMIT);
    return sweep;
}

template <int P>
__global__ void __launch_bounds__(BUILD_THREADS, 1) build_rows_kernel(const BuildArgs args) {
    using Cfg = BuildCfg<P>;
    constexpr int D = Cfg::D, LDX = Cfg::LDX, LDM = Cfg::LDM, LDV = Cfg::LDV, TSZ = Cfg::TSZ;
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
            householder_qr(sX, LDX, m, n, sS);
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
            householder_form_q(sX, LDX, m, kk, sS);
            for (int t = tid; t < m * kk; t += BUILD_THREADS) {
                const int row = t % m, col = t / m;
                Qout[row + (size_t)col * LDX] = sX[row + (size_t)col * LDX];
            }
            __syncthreads();
        }

        // ------------------------------------------------------------------ SVD sweep, right -> left
        double* sM = sR;          // Jacobi operand, row-major [x][a*kprev + y], ld = LDM
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
                sM[(size_t)x * LDM + a * kprev + y] = acc;
                sM0[(size_t)x * LDM + a * kprev + y] = acc;
            }
            __syncthreads();
            double* stage = sX;                 // TSZ doubles: output tensor in fragment order
            double* sV = sX + TSZ;              // [y'][col], ld = LDV: selected right singular vectors
            for (int t = tid; t < TSZ; t += BUILD_THREADS) stage[t] = 0.0;
            double* Aout = env_out + (size_t)c * TSZ;
            if (c == 0) {
                // P-C2 step 3: A_0 (1,2,k_1) = Q_0 Pc; divide by its norm, add log to logscale
                double ss = 0.0;
                for (int t = tid; t < nc; t += BUILD_THREADS) ss += sM[t] * sM[t];
                ss = block_sum(ss, sRed);
                const double s = sqrt(ss);
                if (!(s > 0.0) || !isfinite(s)) { if (tid == 0) raise_flag(args.flags, FLAG_NONFINITE); }
                logs += log(s);
                const double inv_s = 1.0 / s;
                for (int t = tid; t < nc; t += BUILD_THREADS) {
                    const int y = t % kprev, a = t / kprev;
                    stage[env_off(P, 0, a, y)] = sM[t] * inv_s;
                }
                __syncthreads();
                for (int t = tid; t < TSZ; t += BUILD_THREADS) Aout[t] = stage[t];
                __syncthreads();
                break;
            }
            int nrow = ql;
            if (nrow & 1) {   // pad to an even row count with a zero row (never happens for c >= 1)
                for (int t = tid; t < nc; t += BUILD_THREADS) sM[(size_t)nrow * LDM + t] = 0.0;
                ++nrow;
                __syncthreads();
            }
            double fro2 = 0.0;
            for (int t = tid; t < nrow * nc; t += BUILD_THREADS) {
                const double v = sM[(size_t)(t / nc) * LDM + (t % nc)];
                fro2 += v * v;
            }
            fro2 = block_sum(fro2, sRed);
            const double thr2 = fro2 * 1e-30;      // sigma <= 1e-15 |M|_F: below the numerical rank
            jacobi_rows(sM, LDM, nrow, nc, thr2, args.flags);
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
                    sV[(size_t)yp * LDV + col] = v;
                    stage[env_off(P, yp, col / kprev, col % kprev)] = v;
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
