// tnmc_build.cuh -- boundary-MPS environment build (steps a-1..a-7 of DESIGN.md).
//
// One CTA per disorder realisation walks the rows bottom -> top and, per row,
//   A. applies the row MPO (Eq. 7-8) site by site, fused with the left->right
//      canonicalising QR sweep (P-C2 step 1), then
//   B. runs the right->left truncated SVD sweep (P-C2 step 2) and the final scale (P-C2 step 3).
// The MPO tensors are never materialised.  With W[l,a,r,d] = delta(l,a) B_r[a,r] B_d[a,d] the
// product tensor is  A'[(l,i),a,(r,k)] = delta(l,a) B_r[a,r] C_a[i,k],  C_a = sum_m B_d[a,m] A[i,m,k],
// so with the carried factor R = [R_0 | R_1] (column blocks l = 0, 1) the QR operand of a site is
//   X[(x,a),(r,k)] = B_r[a,r] T_a[x,k],  T_a = R_a C_a,   i.e.  X = blockdiag(T_0, T_1) (B_r (x) 1).
// B_r (x) 1 is invertible, so an orthonormal basis of X's columns is blockdiag(Q_0, Q_1) with
// T_a = Q_a R'_a: TWO independent thin QRs of half the size (4x fewer flops, half the depth), run
// side by side by the two halves of the CTA.  The factor pushed right is
// R_new[(a,y),(r,k)] = B_r[a,r] R'_a[y,k] (not triangular -- it need not be: any orthonormal basis
// of the left block is an equally good gauge for the SVD sweep).
// Q_a is never formed: the SVD sweep applies its reflectors to [Pc_a; 0] directly,
//   M = [Q_0 Pc_0 | Q_1 Pc_1]   (Pc = M V_k carried from the site to the right),
// column by column with no barrier between reflectors.
#pragma once
#include "tnmc_common.cuh"
#include "tnmc_linalg.cuh"

namespace tnmc {

struct BuildArgs {
    JView J;
    double beta;
    int L, chi;
    int dis_begin;               // CTA b works on disorder dis_begin + b
    int row_hi, row_lo;          // processes rows row_hi-1, ..., row_lo; row row_hi must be stored
    const int* slot_of_row;      // [L] device: env slot of each row for this pass (-1: not stored)
    EnvRef env;                  // env base (FP64 or FP32 storage)
    size_t env_dis_stride;       // elements per disorder (n_slots * L * 2P^2)
    double* qbuf;                // scratch, per disorder L * QSZ doubles (reflectors of the QR sweep)
    double* m0buf;               // scratch, per disorder D*D doubles (M before rotation; used when P == 32)
    double* logscale;            // (n_dis, L): logscale of every row (written for rows built)
    unsigned long long* flags;
};

template <int P>
struct BuildCfg {
    static constexpr int NT = 8 * P;          // threads per CTA: one quad per column of a 2P-column matrix
    static constexpr int D = 2 * P;           // doubled bond
    static constexpr int LPP = 8;             // lanes per row pair in the Jacobi (8 measured best at chi = 16 and 32, 4 and 2 slower)
    static constexpr int LDX = D + 4;         // column-major leading dim (= 4 mod 16: a half-warp of 4 quads hits 16 distinct 8-byte banks)
    static constexpr int LDM = D + 2;         // row length of the Jacobi operand (row-major)
    static constexpr int LDV = D + 1;         // row length of the selected right singular vectors
    static constexpr int LDR = P + 1;         // row length of the carried R_a[x][i]
    static constexpr int LDU = P + 1;         // row length of the carried Pc[z][y]
    static constexpr int TSZ = 2 * P * P;     // doubles per stored site tensor
    static constexpr int QSZ = LDX * D + 2 * D;   // doubles per site of the reflector scratch: image of X + tau + scale
    // shared-memory carve-up (doubles)
    static constexpr int X_OFF = 0;                       // LDX*D : T_0 | T_1 (QR sweep); M, then stage + V_k (SVD sweep)
    static constexpr int Y_OFF = X_OFF + LDX * D;         // D*LDM >= 2*D*LDR, LDX*D : carried R (QR sweep); reflectors, then Jacobi operand
    static constexpr int Y_SZ = (D * LDM > LDX * D ? D * LDM : LDX * D);
    // M before rotation (needed once more for M V_k) lives in shared memory for P <= 16 and in an
    // L2-resident global scratch for P = 32, which brings the CTA to 88 KB: two CTAs per SM.
    static constexpr bool M0_GLOBAL = P >= 32;
    static constexpr int CTAS_PER_SM = P >= 32 ? 2 : 3;
    static constexpr bool JACOBI_HELD_ROW = P >= 32;     // jacobi_rows4 (measured faster at chi = 32, slower at chi = 16)
    static constexpr int Z_OFF = Y_OFF + Y_SZ;            // D*D   : M before rotation (SVD sweep), P <= 16 only
    static constexpr int U_OFF = Z_OFF + (M0_GLOBAL ? 0 : D * D);   // D*LDU : C_a (QR sweep); carried Pc / M V_k (SVD sweep)
    static constexpr int S_OFF = U_OFF + D * LDU;         // D + 24 + D + 40 : tau / QRCP scratch / sigma / reduction scratch
    static constexpr int N_DBL = S_OFF + 2 * D + 64 + 48 + 40 + D + 8;   // + reflector scales [D] and the QRs' published norms [4]
    static size_t smem_bytes(int L) { return sizeof(double) * N_DBL + sizeof(int) * (L + 2 + 2 * D + 2 + 48); }
};

template <int P>
__global__ void __launch_bounds__(BuildCfg<P>::NT, BuildCfg<P>::CTAS_PER_SM) build_rows_kernel(const BuildArgs args) {
    using Cfg = BuildCfg<P>;
    constexpr int NT = Cfg::NT, HALF = NT / 2, D = Cfg::D, LDX = Cfg::LDX, LDM = Cfg::LDM, LDV = Cfg::LDV,
                  LDR = Cfg::LDR, LDU = Cfg::LDU, TSZ = Cfg::TSZ;
    constexpr int MAXK = P / 2;          // rows per quad lane: every matrix here has at most D = 4 MAXK rows
    extern __shared__ __align__(16) double smem[];
    double* sX = smem + Cfg::X_OFF;
    double* sY = smem + Cfg::Y_OFF;
    double* sA = sX;                     // site tensor staging of the QR sweep (X is free until T is written)
    double* sU = smem + Cfg::U_OFF;
    double* sTau = smem + Cfg::S_OFF;    // [D]  tau of block a at a*P (QR sweep) / of the QRCP
    double* sCn = sTau + D;              // [64 + 8] remaining column norms and per-warp partial sums of the QRCP
    double* sSig = sCn + 72;             // [D]  sigma
    double* sRed = sSig + D;             // [40] block reduction scratch
    double* sScl = sRed + 40;            // [D]  scale of block a's reflectors at a*P (v_j = [1; scale_j x_{i>j}])
    double* sNrm = sScl + D;             // [4]  squared norm of the next pivot column, two per block QR
    int* sq = reinterpret_cast<int*>(smem + Cfg::N_DBL);   // [L+1] rows q_c of the carried R = left bond of Q_c
    int* spos = sq + args.L + 2;                           // [D] rank / position of each Jacobi row
    int* sperm = spos + D;                                 // [D] step at which each column was the QRCP pivot
    int* sNr = sperm + D;                                  // [2] rows of R kept by the QRCP
    unsigned* sWk = reinterpret_cast<unsigned*>(sNr + 2);  // [48] per-warp pivot candidates of the QRCP

    const int tid = threadIdx.x;
    const int half = tid >= HALF ? 1 : 0, gt = tid - half * HALF;
    const int d = args.dis_begin + blockIdx.x;
    const int L = args.L, chi = args.chi;
    const int f32 = args.env.lay32;      // selects the fragment order of the stored tensors
    const double beta = args.beta;
    const size_t env_d = (size_t)d * args.env_dis_stride;
    double* qbuf_d = args.qbuf + (size_t)d * (size_t)L * Cfg::QSZ;
    double* ls_d = args.logscale + (size_t)d * L;
    for (int r = args.row_hi - 1; r >= args.row_lo; --r) {
        const size_t env_in = env_d + (size_t)args.slot_of_row[r + 1] * L * TSZ;
        const size_t env_out = env_d + (size_t)args.slot_of_row[r] * L * TSZ;
        double logs = 0.0;   // all threads carry the same value

        // ------------------------------------------------------------------ A. QR sweep, left -> right
        double* sR = sY;     // carried R_a[x][i] at a*D*LDR, row length LDR
        if (tid == 0) { sq[0] = 1; sR[0] = 1.0; sR[D * LDR] = 1.0; }
        __syncthreads();
        for (int c = 0; c < L; ++c) {
            const int bl = row_bond(L, chi, r + 1, c), br = row_bond(L, chi, r + 1, c + 1);
            const int q = sq[c];
            const size_t Ain = env_in + (size_t)c * TSZ;
            for (int t = tid; t < TSZ; t += NT) sA[t] = args.env.ld(Ain + t);
            __syncthreads();
            {   // C_a[i][k] = sum_m B_d[a][m] A[i][m][k]      (Eq. 7: B_d[a][m] = exp(beta Jd (2a-1)(2m-1)))
                const double jd = args.J.jdv(d, r, c);
                const double w_same = exp(beta * jd), w_diff = exp(-beta * jd);
                for (int t = tid; t < 2 * bl * br; t += NT) {
                    const int k = t % br, i = (t / br) % bl, a = t / (br * bl);
                    sU[(a * P + i) * LDU + k] = w_same * sA[env_off_p(P, i, a, k, f32)] + w_diff * sA[env_off_p(P, i, 1 - a, k, f32)];
                }
            }
            __syncthreads();
            // T_a[x][k] = sum_i R_a[x][i] C_a[i][k]  -> column k of block a of X: a (q x bl)(bl x br) product per spin
            // block on the FP64 tensor pipe; a warp takes 8-row strips (a, x0) and all column tiles of the strip
            {
                const int warp = tid >> 5, lane = tid & 31;
                const int strips = (q + 7) >> 3;
                for (int st = warp; st < 2 * strips; st += NT / 32) {
                    const int a = st / strips, x0 = (st - a * strips) * 8;
                    const double* Ra = sR + (size_t)a * D * LDR;
                    const double* Ca = sU + (size_t)a * P * LDU;
                    double* Xa = sX + (size_t)a * P * LDX;
                    dmma_strip<P / 8>(bl, lane,
                        [&](int g, int i) { return (x0 + g < q && i < bl) ? Ra[(size_t)(x0 + g) * LDR + i] : 0.0; },
                        [&](int i, int k) { return (i < bl && k < br) ? Ca[(size_t)i * LDU + k] : 0.0; },
                        [&](int g, int k, double v) { if (x0 + g < q && k < br) Xa[(size_t)k * LDX + x0 + g] = v; });
                }
            }
            __syncthreads();
            double* Qout = qbuf_d + (size_t)c * Cfg::QSZ;
            if (c == L - 1) {
                // last site (br = 1): not orthogonalised (P-C2 step 1 stops at L-2); T_a[:,0] is column a of its M
                for (int t = tid; t < 2 * q; t += NT) {
                    const int x = t % q, a = t / q;
                    Qout[(size_t)(a * P) * LDX + x] = sX[(size_t)(a * P) * LDX + x];
                }
                if (tid == 0) sq[L] = 1;
                __syncthreads();
                break;
            }
            const int p = q < br ? q : br;
            householder_qr_g<MAXK>(sX + (size_t)half * P * LDX, LDX, q, br, sTau + half * P, sScl + half * P, sNrm + 2 * half, gt, HALF, 1 + half);
            __syncthreads();
            // R_new[(a,y)][(rr,k)] = B_r[a][rr] R'_a[y][k] / |R_new|_F;  logscale += log |R_new|_F
            const double jr = args.J.jrv(d, r, c);
            const double w_same = exp(beta * jr), w_diff = exp(-beta * jr);
            double ss = 0.0;
            for (int t = tid; t < 2 * p * br; t += NT) {
                const int y = t % p, k = (t / p) % br, a = t / (p * br);
                const double v = k >= y ? sX[(size_t)(a * P + k) * LDX + y] : 0.0;
                ss = fma(v, v, ss);
            }
            ss = block_sum(ss, sRed) * (w_same * w_same + w_diff * w_diff);
            const double s = sqrt(ss);
            if (!(s > 0.0) || !isfinite(s)) { if (tid == 0) raise_flag(args.flags, FLAG_NONFINITE); }
            logs += log(s);
            const double inv_s = 1.0 / s;
            for (int t = tid; t < 2 * p * br; t += NT) {
                const int k = t % br, y = (t / br) % p, a = t / (p * br);
                const double v = k >= y ? sX[(size_t)(a * P + k) * LDX + y] * inv_s : 0.0;
                sR[(size_t)a * D * LDR + (size_t)(a * p + y) * LDR + k] = w_same * v;          // rr == a
                sR[(size_t)(1 - a) * D * LDR + (size_t)(a * p + y) * LDR + k] = w_diff * v;    // rr != a
            }
            if (tid == 0) sq[c + 1] = 2 * p;
            // reflectors (below the diagonal of each block) and tau -> scratch for the SVD sweep
            for (int t = tid; t < 2 * q * p; t += NT) {
                const int x = t % q, z = (t / q) % p, a = t / (q * p);
                Qout[(size_t)(a * P + z) * LDX + x] = sX[(size_t)(a * P + z) * LDX + x];
            }
            for (int t = tid; t < 2 * p; t += NT) {
                const int z = t % p, a = t / p;
                Qout[LDX * D + a * P + z] = sTau[a * P + z];
                Qout[LDX * D + D + a * P + z] = sScl[a * P + z];
            }
            __syncthreads();
        }

        // ------------------------------------------------------------------ B. SVD sweep, right -> left
        double* sMj = sY;             // Jacobi operand (rows of R), row-major, row length LDM
        double* sM0 = Cfg::M0_GLOBAL ? args.m0buf + (size_t)d * D * D : smem + Cfg::Z_OFF;   // M before rotation, column-major, leading dim D
        double* stage = sX;           // output tensor in fragment order (once the QRCP result has left X)
        double* sV = sX + TSZ;        // [y'][col], row length LDV: selected right singular vectors
        int kprev = 1;
        for (int c = L - 1; c >= 0; --c) {
            const int q = sq[c];
            const int nc = 2 * kprev;
            const double* Qin = qbuf_d + (size_t)c * Cfg::QSZ;
            if (c == L - 1) {
                for (int t = tid; t < 2 * q; t += NT) {
                    const int x = t % q, a = t / q;
                    sX[(size_t)a * LDX + x] = Qin[(size_t)(a * P) * LDX + x];
                }
            } else {
                // M = [Q_0 Pc_0 | Q_1 Pc_1]: reflectors of block a applied to [Pc_a; 0]
                const int p = sq[c + 1] >> 1;
                // the p reflector columns of a block are contiguous in the scratch image of X: flat copy, four loads in
                // flight per thread (rows >= q of a column were never written and are never read)
                for (int a = 0; a < 2; ++a) {
                    const double* src = Qin + (size_t)a * P * LDX;
                    double* dst = sY + (size_t)a * P * LDX;
                    const int nflat = p * LDX;
                    for (int t = tid; t < nflat; t += 4 * NT) {
                        const int t1 = t + NT, t2 = t + 2 * NT, t3 = t + 3 * NT;
                        const double v0 = src[t];
                        const double v1 = t1 < nflat ? src[t1] : 0.0;
                        const double v2 = t2 < nflat ? src[t2] : 0.0;
                        const double v3 = t3 < nflat ? src[t3] : 0.0;
                        dst[t] = v0;
                        if (t1 < nflat) dst[t1] = v1;
                        if (t2 < nflat) dst[t2] = v2;
                        if (t3 < nflat) dst[t3] = v3;
                    }
                }
                for (int t = tid; t < 2 * p; t += NT) {
                    const int z = t % p, a = t / p;
                    sTau[a * P + z] = Qin[LDX * D + a * P + z];
                    sScl[a * P + z] = Qin[LDX * D + D + a * P + z];
                }
                for (int t = tid; t < q * nc; t += NT) {
                    const int x = t % q, col = t / q;
                    const int a = col / kprev, y = col - a * kprev;
                    sX[(size_t)col * LDX + x] = x < p ? sU[(size_t)(a * p + x) * LDU + y] : 0.0;
                }
                __syncthreads();
                householder_apply_g<MAXK>(sY + (size_t)half * P * LDX, LDX, sTau + half * P, sScl + half * P, q, p,
                                          sX + (size_t)half * kprev * LDX, LDX, kprev, gt, HALF, 1 + half);
            }
            __syncthreads();
            const size_t Aout = env_out + (size_t)c * TSZ;
            if (c == 0) {
                // P-C2 step 3: A_0 (1,2,k_1) = M (1 x nc); divide by its norm, add log to logscale
                double ss = 0.0;
                for (int t = tid; t < nc; t += NT) { const double v = sX[(size_t)t * LDX]; ss = fma(v, v, ss); }
                ss = block_sum(ss, sRed);
                const double s = sqrt(ss);
                if (!(s > 0.0) || !isfinite(s)) { if (tid == 0) raise_flag(args.flags, FLAG_NONFINITE); }
                logs += log(s);
                const double inv_s = 1.0 / s;
                const double m0 = tid < nc ? sX[(size_t)tid * LDX] * inv_s : 0.0;
                __syncthreads();
                for (int t = tid; t < TSZ; t += NT) stage[t] = 0.0;
                __syncthreads();
                if (tid < nc) stage[env_off_p(P, 0, tid / kprev, tid % kprev, f32)] = m0;
                __syncthreads();
                for (int t = tid; t < TSZ; t += NT) args.env.st(Aout + t, stage[t]);
                __syncthreads();
                break;
            }
            for (int t = tid; t < q * nc; t += NT) {
                const int x = t % q, col = t / q;
                sM0[(size_t)col * D + x] = sX[(size_t)col * LDX + x];
            }
            // M = Q (R P^T) with column pivoting, R only and in M's own column order; rows of R below the
            // numerical rank (sigma <= 1e-15 |M|_F) are dropped.  Singular values and right singular
            // vectors of M are those of R P^T.
            int* spst = sperm;                       // step at which each column was the pivot
            const double fro2 = householder_qrcp2<MAXK>(sX, LDX, q, nc, sCn, sWk, spst, sNr);
            const int nrow = *sNr;                   // rows of R kept (even)
            for (int t = tid; t < nrow * D; t += NT) {      // rows zero-padded to D columns for the Jacobi
                const int j = t % D, i = t / D;
                sMj[(size_t)i * LDM + j] = (j < nc && i <= spst[j]) ? sX[i + (size_t)j * LDX] : 0.0;
            }
            __syncthreads();
            const double thr2 = fro2 * 1e-30;      // sigma <= 1e-15 |M|_F: below the numerical rank
            // chi = 32: one row of each pair held in registers, norms carried (jacobi_rows4: C3 build 6.48 -> 5.97 s);
            // chi <= 16: one warp per scheduler, bound by the latency of the dependent chain, where the bookkeeping of
            // the held row costs more than the loads it saves (C2 build 93 -> 100 ms): jacobi_rows2
            constexpr int JNK = (D + 2 * Cfg::LPP - 1) / (2 * Cfg::LPP);
            if (nrow >= 2) {
                static_assert(JNK * 2 * Cfg::LPP < LDM, "the carried norm of a row lives in the spare column after its padded width");
                if constexpr (Cfg::JACOBI_HELD_ROW) jacobi_rows4<JNK, Cfg::LPP>(sMj, LDM, JNK * 2 * Cfg::LPP, nrow, fro2, thr2, args.flags);
                else jacobi_rows2<JNK, Cfg::LPP>(sMj, LDM, nrow, fro2, thr2, args.flags);
            }
            // singular values = row norms
            {
                const int grp = tid >> 3, t8 = tid & 7;
                for (int x = grp; x < nrow; x += (NT >> 3)) {
                    double a = 0.0;
                    for (int cc = t8; cc < nc; cc += 8) { const double v = sMj[(size_t)x * LDM + cc]; a = fma(v, v, a); }
#pragma unroll
                    for (int o = 4; o > 0; o >>= 1) a += __shfl_xor_sync(0xffu << ((tid & 31) & ~7), a, o);
                    if (t8 == 0) sSig[x] = sqrt(a);
                }
            }
            int k = chi < q ? chi : q;
            if (nc < k) k = nc;
            for (int t = tid; t < TSZ; t += NT) stage[t] = 0.0;
            if (k > nrow) {    // kept directions beyond the numerical rank stay zero rows
                for (int t = tid; t < (k - nrow) * LDV; t += NT) sV[(size_t)nrow * LDV + t] = 0.0;
                if (tid == 0) raise_flag(args.flags, FLAG_SIGMA_ZERO);
            }
            __syncthreads();
            for (int x = tid; x < nrow; x += NT) {
                const double sx = sSig[x];
                int rank = 0;
                for (int y = 0; y < nrow; ++y) {
                    const double sy = sSig[y];
                    rank += (sy > sx) || (sy == sx && y < x);
                }
                spos[x] = rank < k ? rank : -1;
                if (rank < k && !(sx * sx > thr2)) raise_flag(args.flags, FLAG_SIGMA_ZERO);
            }
            __syncthreads();
            // A_c[y'][a][y] = v_{y'}  (rows of V_k^T), staged in fragment order and as plain rows
            for (int t = tid; t < nrow * nc; t += NT) {
                const int col = t % nc, x = t / nc;
                const int yp = spos[x];
                if (yp >= 0) {
                    const double sx = sSig[x];
                    // a kept direction below the numerical rank carries no weight (M v = 0 for any
                    // orthonormal completion); it is stored as a zero row
                    const double v = sx * sx > thr2 ? sMj[(size_t)x * LDM + col] / sx : 0.0;
                    sV[(size_t)yp * LDV + col] = v;     // col = (a, y) = a * kprev + y
                    stage[env_off_p(P, yp, col / kprev, col % kprev, f32)] = v;
                }
            }
            __syncthreads();
            for (int t = tid; t < TSZ; t += NT) args.env.st(Aout + t, stage[t]);
            // Pc_next[x][y'] = sum_col M[x][col] V_k[col][y']   (= M V_k, projector form of P-C2 step 2): a (q x nc)(nc x k)
            // product on the FP64 tensor pipe, one 8-row strip of M per warp (M is read once, from L2 at chi = 32)
            {
                const int warp = tid >> 5, lane = tid & 31;
                for (int x0 = 8 * warp; x0 < q; x0 += 8 * (NT / 32)) {
                    dmma_strip<P / 8>(nc, lane,
                        [&](int g, int col) { return (x0 + g < q && col < nc) ? sM0[(size_t)col * D + x0 + g] : 0.0; },
                        [&](int col, int yp) { return (col < nc && yp < k) ? sV[(size_t)yp * LDV + col] : 0.0; },
                        [&](int g, int yp, double v) { if (x0 + g < q && yp < k) sU[(size_t)(x0 + g) * LDU + yp] = v; });
                }
            }
            __syncthreads();
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
__global__ void bottom_row_kernel(JView J, double beta, int L, int P, EnvRef env, size_t env_dis_stride,
                                  int slot, double* logscale) {
    const int c = blockIdx.x, d = blockIdx.y;
    const int TSZ = 2 * P * P;
    const size_t A = (size_t)d * env_dis_stride + ((size_t)slot * L + c) * TSZ;
    for (int t = threadIdx.x; t < TSZ; t += blockDim.x) env.st(A + t, 0.0);
    __syncthreads();
    if (threadIdx.x < 8) {
        const int l = threadIdx.x >> 2, a = (threadIdx.x >> 1) & 1, b = threadIdx.x & 1;
        const double jr = (c == L - 1) ? 0.0 : J.jrv(d, L - 1, c);
        const double bm = exp(beta * jr * (2 * a - 1) * (2 * b - 1));
        if (c == 0) { if (l == 0) env.st(A + env_off_p(P, 0, a, b, env.lay32), bm); }
        else if (c == L - 1) { if (b == 0 && l == a) env.st(A + env_off_p(P, l, a, 0, env.lay32), 1.0); }
        else if (l == a) env.st(A + env_off_p(P, l, a, b, env.lay32), bm);
    }
    if (c == 0 && threadIdx.x == 0) logscale[(size_t)d * L + (L - 1)] = 0.0;
}

// ---------------------------------------------------------------------------------------------
// log Z read-out (a-7; Eq. 6): log Z = logscale_0 + log |sum_sigma Psihat_0(sigma)|,
// the sum taken as the product over c of sum_a A_c[:,a,:] with a running max-abs rescale.
// One warp per disorder; lane j carries component j of the running row vector.
// ---------------------------------------------------------------------------------------------
__global__ void logz_kernel(int L, int chi, int P, int n_dis, EnvRef env, size_t env_dis_stride,
                            int slot0, const double* logscale, double* logZ, unsigned long long* flags) {
    const int d = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (d >= n_dis) return;
    const int lane = threadIdx.x & 31;
    const int TSZ = 2 * P * P;
    const size_t row = (size_t)d * env_dis_stride + (size_t)slot0 * L * TSZ;
    double v = lane == 0 ? 1.0 : 0.0;   // component `lane` of the running vector (P <= 32)
    double lg = logscale[(size_t)d * L];
    for (int c = 0; c < L; ++c) {
        const size_t A = row + (size_t)c * TSZ;
        const int bl = row_bond(L, chi, 0, c), br = row_bond(L, chi, 0, c + 1);
        double acc = 0.0;
        for (int i = 0; i < bl; ++i) {
            const double vi = __shfl_sync(0xffffffffu, v, i);
            if (lane < br) acc += vi * (env.ld(A + env_off_p(P, i, 0, lane, env.lay32)) + env.ld(A + env_off_p(P, i, 1, lane, env.lay32)));
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
        // bonds across the open boundary do not exist (Jr at c = L-1, Jd at r = L-1): masked out whatever the caller put there
        const int8_t jr = c + 1 < L ? Jr[dr * L + c] : (int8_t)0;
        const int8_t jd = (int)(dr % L) + 1 < L ? Jd[dr * L + c] : (int8_t)0;
        rn |= (uint32_t)(jr < 0) << b; rz |= (uint32_t)(jr != 0) << b;
        dn |= (uint32_t)(jd < 0) << b; dz |= (uint32_t)(jd != 0) << b;
    }
    masks[0 * n_words + idx] = rn;
    masks[1 * n_words + idx] = rz;
    masks[2 * n_words + idx] = dn;
    masks[3 * n_words + idx] = dz;
}

// Export one stored row in the paper's layout (L, chi, 2, chi) -- test/inspection hook.
__global__ void export_row_kernel(int L, int chi, int P, EnvRef env, size_t row, double* out) {
    const int c = blockIdx.x;
    const int TSZ = 2 * P * P;
    for (int t = threadIdx.x; t < chi * 2 * chi; t += blockDim.x) {
        const int j = t % chi, a = (t / chi) & 1, i = t / (2 * chi);
        out[(size_t)c * chi * 2 * chi + t] = env.ld(row + (size_t)c * TSZ + env_off_p(P, i, a, j, env.lay32));
    }
}

}  // namespace tnmc
