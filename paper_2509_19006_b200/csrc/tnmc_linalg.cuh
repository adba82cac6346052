// tnmc_linalg.cuh -- shared-memory dense kernels of the compression step (a-4, a-5): Householder QR,
// application of Q from its reflectors, Householder QR with column pivoting and one-sided Jacobi SVD,
// for matrices of at most 64 x 64 doubles.  Everything here is a chain of small dependent steps; the
// design rule is: at most one barrier per serial step, every trailing column handled by a quad of lanes
// (every row pair by a group of lanes) with its loads batched in registers, square roots and divisions
// replaced by MUFU-seeded rsqrt / reciprocal and kept off the critical path where possible.
// (A one-lane-per-column, one-warp variant without any block barrier was measured and is slower: its
// loops wait on shared-memory latency, profiles/r1e notes.)
#pragma once
#include "tnmc_common.cuh"

namespace tnmc {

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

// 1/sqrt(x) and 1/x for normal positive-range doubles without the library routines' special-case
// handling: the MUFU seed (relative error <= 2^-22) and two Newton steps (error squared each time,
// ~1 ulp at the end).  x must be finite, normal and (for rsqrt) positive -- true for every squared
// norm and pivot that reaches them (zeros are excluded by the callers).
__device__ __forceinline__ double fast_rsqrt(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double hx = 0.5 * x;
    r = r * fma(-hx * r, r, 1.5);
    r = r * fma(-hx * r, r, 1.5);
    return r;
}
// one Newton step: relative error ~ 1e-13.  Enough for the Jacobi rotation: an error in w scales both rows of the
// pair alike (directions unchanged), an error in h tilts the angle by 1e-13 of itself (left to the next sweep).
__device__ __forceinline__ double fast_rsqrt1(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double hx = 0.5 * x;
    r = r * fma(-hx * r, r, 1.5);
    return r;
}
__device__ __forceinline__ double fast_rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(r, fma(-x, r, 1.0), r);
    r = fma(r, fma(-x, r, 1.0), r);
    return r;
}

// Quad-cooperative column kernels used by the Householder routines.  A quad (4 lanes, rg = lane & 3)
// owns one column; lane rg handles rows i0 + rg + 4k.  MAXK = max rows per lane.  Loads are batched
// into registers (independent accumulators) so that shared-memory latency overlaps.
template <int MAXK>
__device__ __forceinline__ double quad_dot_update(const double* __restrict__ v, double* __restrict__ col,
                                                  int i0, int m, int rg, unsigned qmask, double tau, double head,
                                                  double& below2) {
    // w = tau * (head + sum_{i >= i0} v_i col_i);  col_i -= w v_i;  below2 = sum_{i >= i0} col_i^2 (after update)
    double x[MAXK], vv[MAXK];
    double w0 = 0.0, w1 = 0.0, w2 = 0.0, w3 = 0.0;
#pragma unroll
    for (int k = 0; k < MAXK; ++k) {
        const int i = i0 + rg + 4 * k;
        const bool in = i < m;
        x[k] = in ? col[i] : 0.0;
        vv[k] = in ? v[i] : 0.0;
    }
#pragma unroll
    for (int k = 0; k < MAXK; k += 4) {
        w0 = fma(vv[k], x[k], w0);
        if (k + 1 < MAXK) w1 = fma(vv[k + 1], x[k + 1], w1);
        if (k + 2 < MAXK) w2 = fma(vv[k + 2], x[k + 2], w2);
        if (k + 3 < MAXK) w3 = fma(vv[k + 3], x[k + 3], w3);
    }
    double w = (w0 + w1) + (w2 + w3);
    w += __shfl_xor_sync(qmask, w, 1);
    w += __shfl_xor_sync(qmask, w, 2);
    w = (w + head) * tau;
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int k = 0; k < MAXK; ++k) {
        const int i = i0 + rg + 4 * k;
        if (i < m) {
            const double nv = fma(-w, vv[k], x[k]);
            col[i] = nv;
            if (k & 1) s1 = fma(nv, nv, s1); else s0 = fma(nv, nv, s0);
        }
    }
    below2 = s0 + s1;
    return w;
}

// The number of live rows shrinks as the factorization proceeds: pick the smallest unrolled depth (a quarter,
// a half, three quarters or all of MAXK rows per lane) that covers rows i0 .. m-1.  The choice is uniform over the
// CTA (m and i0 are), so no divergence; it removes on average half of the predicated loads and FMAs of a sweep.
template <int MAXK>
__device__ __forceinline__ double quad_dot_update_n(const double* __restrict__ v, double* __restrict__ col,
                                                    int i0, int m, int rg, unsigned qmask, double tau, double head,
                                                    double& below2) {
    const int rows = m - i0;
    if (MAXK >= 4) {
        if (rows <= MAXK) return quad_dot_update<(MAXK + 3) / 4>(v, col, i0, m, rg, qmask, tau, head, below2);
        if (rows <= 2 * MAXK) return quad_dot_update<MAXK / 2>(v, col, i0, m, rg, qmask, tau, head, below2);
        if (rows <= 3 * MAXK) return quad_dot_update<(3 * MAXK) / 4>(v, col, i0, m, rg, qmask, tau, head, below2);
    }
    return quad_dot_update<MAXK>(v, col, i0, m, rg, qmask, tau, head, below2);
}

// The same update with the UNSCALED pivot column pc (the reflector vector is pc * scale below row j) and the scalars
// (tau, scale) applied on the fly: w = tau (cj + scale * sum_i pc_i col_i), col_i -= w scale pc_i, row j -> cj - w.
// Returns the squared norm of the updated rows below j (summed over the quad).
template <int K, bool NORM = true>
__device__ __forceinline__ double quad_pivot_update(const double* __restrict__ pc, double* __restrict__ col,
                                                    int j, int m, int rg, unsigned qmask, double tau, double scale) {
    double x[K], vv[K];
    double w0 = 0.0, w1 = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int i = j + 1 + rg + 4 * k;
        const bool in = i < m;
        x[k] = in ? col[i] : 0.0;
        vv[k] = in ? pc[i] : 0.0;
    }
    const double cj = col[j];
#pragma unroll
    for (int k = 0; k < K; k += 2) {
        w0 = fma(vv[k], x[k], w0);
        if (k + 1 < K) w1 = fma(vv[k + 1], x[k + 1], w1);
    }
    double dot = w0 + w1;
    dot += __shfl_xor_sync(qmask, dot, 1);
    dot += __shfl_xor_sync(qmask, dot, 2);
    const double w = tau * fma(scale, dot, cj);
    const double ws = w * scale;
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int i = j + 1 + rg + 4 * k;
        if (i < m) {
            const double nv = fma(-ws, vv[k], x[k]);
            col[i] = nv;
            if (NORM) { if (k & 1) s1 = fma(nv, nv, s1); else s0 = fma(nv, nv, s0); }
        }
    }
    double below2 = s0 + s1;
    if (NORM) {
        below2 += __shfl_xor_sync(qmask, below2, 1);
        below2 += __shfl_xor_sync(qmask, below2, 2);
    }
    if (rg == 0) col[j] = cj - w;
    return below2;
}
template <int MAXK, bool NORM = true>
__device__ __forceinline__ double quad_pivot_update_n(const double* __restrict__ pc, double* __restrict__ col,
                                                      int j, int m, int rg, unsigned qmask, double tau, double scale) {
    const int rows = m - j - 1;
    if (MAXK >= 4) {
        if (rows <= MAXK) return quad_pivot_update<(MAXK + 3) / 4, NORM>(pc, col, j, m, rg, qmask, tau, scale);
        if (rows <= 2 * MAXK) return quad_pivot_update<MAXK / 2, NORM>(pc, col, j, m, rg, qmask, tau, scale);
        if (rows <= 3 * MAXK) return quad_pivot_update<(3 * MAXK) / 4, NORM>(pc, col, j, m, rg, qmask, tau, scale);
    }
    return quad_pivot_update<MAXK, NORM>(pc, col, j, m, rg, qmask, tau, scale);
}

// Reflector from alpha = x_j and nrm2 = sum_{i >= j} x_i^2 (the diagonal entry included, so no
// cancellation): beta = -sign(alpha) sqrt(nrm2), tau = (beta - alpha) / beta, v_i = x_i / (alpha - beta).
__device__ __forceinline__ void reflector_from_norm(double alpha, double nrm2, double& beta, double& tau, double& scale) {
    beta = alpha; tau = 0.0; scale = 0.0;
    if (nrm2 > 1e-280) {   // (smaller: the column is numerically zero against anything it could matter to)
        // one rsqrt and one reciprocal on the critical path (sqrt + two divisions cost 340 cycles on B200)
        const double r = fast_rsqrt(nrm2);
        const double nrm = nrm2 * r;
        const bool pos = alpha >= 0.0;
        beta = pos ? -nrm : nrm;
        tau = (beta - alpha) * (pos ? -r : r);
        scale = fast_rcp(alpha - beta);
    }
}

// ---------------------------------------------------------------------------------------------
// Group versions: the CTA is split into thread groups (multiples of a warp) that each factor their
// own matrix and synchronise on their own named barrier, so two factorizations of one site run
// side by side without meeting at a CTA-wide barrier.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void group_bar(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(nthreads) : "memory");
}

// Householder QR of the m x n column-major X (leading dim ld) by a group of gn threads (thread gt of the group;
// gn/4 >= n - 1 quads, m <= 4 * MAXK).  One barrier per reflector, and nothing serial between barriers: the reflector
// is kept UNSCALED (v_j = [1; scale_j * x_{i>j}] with x the column as it stands) and its scalars (beta, tau, scale) are
// derived by every thread from the diagonal entry and the column's remaining squared norm, which the quad that owns
// column j+1 sums inside its update of step j and publishes before the barrier -- so the rsqrt / reciprocal chain runs
// beside the loads of the dot product instead of in front of 31 waiting quads, and there is no scaling pass over the
// column.  (Round 1 built reflector j+1 in one quad between the update and the barrier: 13.7 % of the kernel's warp
// samples sat at that barrier, profiles/r2c_build32_c3q.md.)
// On return: R on and above the diagonal of X; below the diagonal of column j the unscaled reflector entries;
// tau[j], scl[j] its scalars.  nrm: 2 doubles of scratch.  The caller synchronises before reading X.
template <int MAXK>
__device__ void householder_qr_g(double* X, int ld, int m, int n, double* tau, double* scl, double* nrm, int gt, int gn, int bar) {
    const int kk = m < n ? m : n;
    const int lane = gt & 31;
    const int rg = lane & 3;
    const unsigned qmask = 0xfu << (lane & ~3);
    const int colidx = gt >> 2;
    if (gt < 32) {     // squared norm of column 0 (first warp of the group)
        double ss = 0.0;
        for (int i = lane; i < m; i += 32) { const double v = X[i]; ss = fma(v, v, ss); }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
        if (lane == 0) nrm[0] = ss;
    }
    group_bar(bar, gn);
    for (int j = 0; j < kk; ++j) {
        const double* pc = X + (size_t)j * ld;
        double bet, t, scale;
        reflector_from_norm(pc[j], nrm[j & 1], bet, t, scale);
        const int jj = j + 1 + colidx;
        if (jj < n) {
            double* col = X + (size_t)jj * ld;
            const double below2 = quad_pivot_update_n<MAXK>(pc, col, j, m, rg, qmask, t, scale);
            if (colidx == 0 && rg == 0) nrm[(j + 1) & 1] = below2;     // rows j+1.. of column j+1: the next reflector's norm
        }
        if (gt == 0) { tau[j] = t; scl[j] = scale; }
        group_bar(bar, gn);
        if (gt == 0) X[(size_t)j * ld + j] = bet;     // diagonal of R (column j is read by nobody from here on)
    }
}

// B <- Q B for the m x nb column-major B (leading dim ldb), Q = H_0 H_1 ... H_{kk-1} given by the unscaled
// reflectors below the diagonal of V (leading dim ldv; v_j = [1; scl[j] * V_{i>j, j}]) and tau, without ever forming
// Q.  One quad per column of B (gn/4 >= nb); the columns are independent: no barrier.
template <int MAXK>
__device__ void householder_apply_g(const double* V, int ldv, const double* tau, const double* scl, int m, int kk,
                                    double* B, int ldb, int nb, int gt, int gn, int bar) {
    const int lane = gt & 31;
    const int rg = lane & 3;
    const unsigned qmask = 0xfu << (lane & ~3);
    const int colidx = gt >> 2;
    if (colidx < nb) {
        double* col = B + (size_t)colidx * ldb;
        for (int j = kk - 1; j >= 0; --j) {
            quad_pivot_update_n<MAXK, false>(V + (size_t)j * ldv, col, j, m, rg, qmask, tau[j], scl[j]);
            __syncwarp(qmask);
        }
    }
    (void)gn; (void)bar;
}

// Householder QR with column pivoting, R only, second version: one barrier per step, no column swaps.
//   X (m x n, column-major, leading dim ld; m <= 4 MAXK, n <= blockDim/4) is overwritten by R in
//   PHYSICAL column order: after the call, entry (i, col) of R P^T is X[i + col*ld] for
//   i <= pstep[col] and 0 below (pstep[col] = step at which col was the pivot, or the number of
//   steps done if it never was).  M = Q R P^T, so the rows of this matrix have the singular values
//   and right singular vectors of M in M's own column coordinates -- nothing is permuted back.
//   * Every quad owns a column and keeps its remaining squared norm, summed afresh inside every
//     update (exact, no downdating).  Each warp reduces its columns to (max, index), writes the
//     pair to shared memory, and after the step's single barrier every thread reads the <= 8 pairs
//     and derives the same pivot and the same reflector scalars redundantly.
//   * The reflector is never stored (R only): the pivot column is read as is and its scale is
//     folded into the update, so the dot product runs beside the rsqrt/reciprocal chain.
//   * Steps stop early (at an even step j) once (n - j) * max remaining norm^2 <= 1e-30 |X|_F^2:
//     every further row of R is below the numerical rank (sigma <= 1e-15 |X|_F) and is dropped.
//   Returns |X|_F^2; *n_rows_out = rows of R kept (even).
template <int MAXK>
__device__ double householder_qrcp2(double* X, int ld, int m, int n, double* cn, unsigned* wk, int* pstep, int* n_rows_out) {
    // cn: [8] per-warp partial sums at cn + 64;  wk: [2][3][8] per-warp (norm pattern high, low, column)
    const int kk = m < n ? m : n;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int rg = lane & 3;
    const unsigned qmask = 0xfu << (lane & ~3);
    const int cq = threadIdx.x >> 2;
    const bool has_col = cq < n;
    double* col = X + (size_t)(has_col ? cq : 0) * ld;
    double* wsum = cn + 64;
    bool active = has_col;
    double myn = 0.0;
    if (has_col) {
        double s0 = 0.0, s1 = 0.0;
        for (int i = rg; i < m; i += 8) {
            const double a = col[i]; s0 = fma(a, a, s0);
            if (i + 4 < m) { const double b = col[i + 4]; s1 = fma(b, b, s1); }
        }
        double ss = s0 + s1;
        ss += __shfl_xor_sync(qmask, ss, 1);
        ss += __shfl_xor_sync(qmask, ss, 2);
        myn = ss;
    }
    // |X|_F^2: per-warp partial sums (each column counted once, by its rg == 0 lane), fixed order
    {
        double part = (has_col && rg == 0) ? myn : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if (lane == 0) wsum[warp] = part;
    }
    // Pivot search: a non-negative double orders like its 64-bit pattern, so the warp's largest remaining
    // norm comes from two redux.sync.max (high word, then low word among the lanes that tie on the high
    // word) and a redux.sync.min on the column index among exact ties; lane 0 publishes (pattern, column).
    // After the barrier every thread scans the <= 8 published pairs: exact argmax, smallest column on ties.
    auto publish = [&](int buf) {
        const unsigned hi = active ? (unsigned)__double2hiint(myn) + 1u : 0u;     // +1: an active zero column beats an inactive one
        const unsigned lo = (unsigned)__double2loint(myn);
        const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
        const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
        const unsigned mc = __reduce_min_sync(0xffffffffu, (hi == mh && lo == ml) ? (unsigned)cq : 0xffffu);
        if (lane == 0) { wk[buf * 24 + warp] = mh; wk[buf * 24 + 8 + warp] = ml; wk[buf * 24 + 16 + warp] = mc; }
    };
    publish(0);
    __syncthreads();
    double fro2 = 0.0;
    for (int w = 0; w < nw; ++w) fro2 += wsum[w];
    const double thr2 = fro2 * 1e-30;
    int my_pstep = kk;
    double pend_beta = 0.0;
    int j = 0;
    for (; j < kk; ++j) {
        const int buf = j & 1;
        // second level of the same reduction: lane w < nw takes warp w's candidate, three redux over the warp
        const unsigned ch = lane < nw ? wk[buf * 24 + lane] : 0u;
        const unsigned cl = lane < nw ? wk[buf * 24 + 8 + lane] : 0u;
        const unsigned cc = lane < nw ? wk[buf * 24 + 16 + lane] : 0xffffu;
        const unsigned mh = __reduce_max_sync(0xffffffffu, ch);
        const unsigned ml = __reduce_max_sync(0xffffffffu, ch == mh ? cl : 0u);
        const unsigned mc = __reduce_min_sync(0xffffffffu, (ch == mh && cl == ml) ? cc : 0xffffu);
        const int bi = mh != 0u ? (int)mc : 0;
        const double best = mh != 0u ? __hiloint2double((int)(mh - 1u), (int)ml) : 0.0;
        if ((j & 1) == 0 && !(best * (double)(n - j) > thr2)) break;
        const double* pc = X + (size_t)bi * ld;
        double bet, tau, scale;
        if (active && cq != bi) {
            // dot product with the unscaled pivot column; the scalars are folded in on the fly
            reflector_from_norm(pc[j], best, bet, tau, scale);
            const double below2 = quad_pivot_update_n<MAXK>(pc, col, j, m, rg, qmask, tau, scale);
            myn = below2;
        } else if (active) {   // this quad owns the pivot: its column is final (row j becomes beta, written after the barrier)
            reflector_from_norm(pc[j], best, bet, tau, scale);
            pend_beta = bet;
            my_pstep = j;
            active = false;
        }
        publish(buf ^ 1);
        __syncthreads();
        if (my_pstep == j && has_col && rg == 0) col[j] = pend_beta;
    }
    if (has_col && rg == 0) pstep[cq] = my_pstep < j ? my_pstep : j;
    *n_rows_out = j;
    __syncthreads();
    return fro2;
}

// One-sided (Hestenes) Jacobi on the rows of M, second version: as jacobi_rows, but a pair's two
// squared norms are summed together with its dot product from the registers that hold the rows
// (three sums share the three shuffle stages), so nothing is cached in shared memory, nothing is
// updated after a rotation and nothing is refreshed per sweep; and the rotation comes from two FP64
// rsqrt with no division and no FP32 detour:
//   d = b - a, h = sqrt(d^2 + 4 g^2), u = |d| + h, w = 1 / sqrt(u^2 + 4 g^2), cos = u w, sin = sign(d) 2 g w.
// The caller zero-pads every row to the full 2 LPP NK columns (rotations keep zeros zero).
// All n rows take part (n even); rows at or below thr2 are left alone.  A sweep is the last one when every pair it
// met had |cos| <= 1e-6 BEFORE its rotation (the rotation is still applied: quadratic convergence leaves ~1e-12, two
// orders below the 1e-10 the parity needs; 1e-8 measured the same deviations from the oracle on all of C2 and 2 % more time).
// The test is purely relative: every kept row v enters M V_k V_k^T, so a row of tiny sigma that is left at an
// angle eps from a dominant row changes the state by eps * sigma_1, whatever its own sigma.  (Round 1 also let a
// sweep end when |g| <= 256 eps |M|_F max(|x|,|y|); on C2 beta = 2 -- kept sigma down to 1e-15 sigma_1 -- that left
// conditionals of 4 of the 100 disorders 1e-7..5e-6 from the oracle; with the relative test the worst is 7e-9,
// log Z 2e-13; cost: C2 build +3 %, C3 build +4.7 %.)  LPP lanes per row pair (a power of
// two <= 8), NK = ceil(max nc / (2 LPP)) column pairs per lane.  Returns the sweeps done.
template <int NK, int LPP>
__device__ int jacobi_rows2(double* M, int ld, int n, double fro2, double thr2, unsigned long long* flags) {
    const int grp = threadIdx.x / LPP, t8 = threadIdx.x % LPP;
    const int npairs = n >> 1;
    (void)fro2;
    const unsigned gmask = ((1u << LPP) - 1u) << ((threadIdx.x & 31) & ~(LPP - 1));
    const double rot2 = 256.0 * 4.930380657631324e-32;             // (16 eps)^2
    const double big2 = 1e-12;                                     // (1e-6)^2
    const int c0 = 2 * t8;                                         // this lane's columns: c0 + 2 LPP k, c0 + 2 LPP k + 1
    int sweep = 0;
    for (; sweep < 60; ++sweep) {
        int big = 0;
        // round-robin (circle) schedule: pair 0 is (n-1, round), pair p >= 1 is ((round + p) mod (n-1),
        // (round - p) mod (n-1)); both members advance by one per round
        int q1 = grp, q2 = grp == 0 ? 0 : n - 1 - grp;
        for (int round = 0; round < n - 1; ++round) {
            if (grp < npairs) {
                int r1 = grp == 0 ? n - 1 : q1, r2 = q2;
                if (++q1 == n - 1) q1 = 0;
                if (++q2 == n - 1) q2 = 0;
                if (r1 > r2) { const int t = r1; r1 = r2; r2 = t; }
                double* x = M + (size_t)r1 * ld;
                double* y = M + (size_t)r2 * ld;
                double2 xv[NK], yv[NK];
#pragma unroll
                for (int k = 0; k < NK; ++k) {      // rows are zero-padded to the full 2 LPP NK columns: no bounds checks
                    const int c = c0 + 2 * LPP * k;
                    xv[k] = *reinterpret_cast<const double2*>(x + c);
                    yv[k] = *reinterpret_cast<const double2*>(y + c);
                }
                double a = 0.0, b = 0.0, g = 0.0, a1 = 0.0, b1 = 0.0, g1 = 0.0;
#pragma unroll
                for (int k = 0; k < NK; ++k) {
                    a = fma(xv[k].x, xv[k].x, a);  a1 = fma(xv[k].y, xv[k].y, a1);
                    b = fma(yv[k].x, yv[k].x, b);  b1 = fma(yv[k].y, yv[k].y, b1);
                    g = fma(xv[k].x, yv[k].x, g);  g1 = fma(xv[k].y, yv[k].y, g1);
                }
                a += a1; b += b1; g += g1;
#pragma unroll
                for (int o = LPP / 2; o > 0; o >>= 1) {
                    a += __shfl_xor_sync(gmask, a, o);
                    b += __shfl_xor_sync(gmask, b, o);
                    g += __shfl_xor_sync(gmask, g, o);
                }
                const double g2 = g * g, ab = a * b;
                if (a > thr2 && b > thr2 && g2 > rot2 * ab) {
                    big |= g2 > big2 * ab;
                    const double dd = b - a;
                    const double g24 = 4.0 * g2;
                    const double h2 = fma(dd, dd, g24);
                    const double u = fabs(dd) + h2 * fast_rsqrt1(h2);
                    const double w = fast_rsqrt1(fma(u, u, g24));
                    const double cs = u * w;
                    double sn = 2.0 * g * w;
                    if (dd < 0.0) sn = -sn;
#pragma unroll
                    for (int k = 0; k < NK; ++k) {
                        const int c = c0 + 2 * LPP * k;
                        double2 xn, yn;
                        xn.x = fma(cs, xv[k].x, -sn * yv[k].x);  yn.x = fma(sn, xv[k].x, cs * yv[k].x);
                        xn.y = fma(cs, xv[k].y, -sn * yv[k].y);  yn.y = fma(sn, xv[k].y, cs * yv[k].y);
                        *reinterpret_cast<double2*>(x + c) = xn;
                        *reinterpret_cast<double2*>(y + c) = yn;
                    }
                }
            }
            __syncthreads();
        }
        if (!__syncthreads_or(big)) { ++sweep; break; }
    }
    if (sweep >= 60 && threadIdx.x == 0) raise_flag(flags, FLAG_JACOBI_LIMIT);
    return sweep;
}

// One-sided Jacobi with a HELD ROW (used at chi = 32).  The same round-robin schedule as jacobi_rows2 (round R of a
// sweep holds the pairs (R + p, R - p) mod (n-1), p = 1 .. n/2 - 1, and (n-1, R)), but the pairs are dealt to the
// lane groups so that one row of every pair STAYS IN THE GROUP'S REGISTERS from round to round.  In the circle
// method a row is the "plus" member of pairs p = n/2-1, ..., 1, then meets row n-1, then is the "minus" member of
// p = 1, ..., n/2-1: a group adopts a row when it turns plus, keeps it for n/2 rounds, and writes it back after it
// has met row n-1; only the partner row (a minus member, or row n-1) goes through shared memory each round: half
// the shared-memory traffic of a round.  The rotation is written symmetrically (new r = cos r -+ sin r') so it does
// not depend on which member is held.
// The squared row norms are CARRIED instead of re-summed every round: a rotation by the Jacobi angle changes them
// by exactly -+ t g (t = tan, g = the pair's dot product; the larger grows, the smaller shrinks, by 2 g^2 / u), so
// a round sums one dot product instead of three.  The held row's norm travels in a register, a moving row's norm in
// the spare column `nslot` of its shared-memory row (nslot >= the padded width, < ld); all norms are summed afresh
// at the start of every sweep, so the carried values are at most n-1 updates (a few 1e-15 relative) old -- they
// only steer the rotation angle and the thresholds; the singular values are summed from the rows afterwards.
// Otherwise the same arguments, thresholds and return value as jacobi_rows2.
template <int NK, int LPP>
__device__ int jacobi_rows4(double* M, int ld, int nslot, int n, double fro2, double thr2, unsigned long long* flags) {
    const int grp = threadIdx.x / LPP, t8 = threadIdx.x % LPP;
    const int m = n >> 1, n1 = n - 1;
    const bool act = grp < m;
    (void)fro2;
    const unsigned gmask = ((1u << LPP) - 1u) << ((threadIdx.x & 31) & ~(LPP - 1));
    const double rot2 = 256.0 * 4.930380657631324e-32;             // (16 eps)^2
    const double big2 = 1e-12;                                     // (1e-6)^2
    const int c0 = 2 * t8;
    int sweep = 0;
    for (; sweep < 60; ++sweep) {
        int big = 0;
        // state of this group at round 0: age = rounds since it adopted its row, delta = m - 1 - age = the p of
        // its pair (0: the row meets row n-1); own = delta, pm = (round - delta) mod (n-1) = the minus member
        int age = grp == 0 ? 0 : m - grp;
        int own = m - 1 - age;
        int pm = own == 0 ? 0 : n1 - own;
        double2 ov[NK];
        double ao = 0.0;     // carried squared norm of the held row
        if (act) {           // fresh norms of rows 2 grp, 2 grp + 1 into their slots
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double* x = M + (size_t)(2 * grp + h) * ld;
                double s0 = 0.0, s1 = 0.0;
#pragma unroll
                for (int k = 0; k < NK; ++k) {
                    const double2 v = *reinterpret_cast<const double2*>(x + c0 + 2 * LPP * k);
                    s0 = fma(v.x, v.x, s0);  s1 = fma(v.y, v.y, s1);
                }
                s0 += s1;
#pragma unroll
                for (int o = LPP / 2; o > 0; o >>= 1) s0 += __shfl_xor_sync(gmask, s0, o);
                if (t8 == 0) M[(size_t)(2 * grp + h) * ld + nslot] = s0;
            }
        }
        __syncthreads();
        if (act) {
#pragma unroll
            for (int k = 0; k < NK; ++k) ov[k] = *reinterpret_cast<const double2*>(M + (size_t)own * ld + c0 + 2 * LPP * k);
            ao = M[(size_t)own * ld + nslot];
        }
        for (int round = 0; round < n1; ++round) {
            if (act) {
                const bool last = age == m - 1;                    // delta == 0: partner is row n-1
                const int prt = last ? n1 : pm;
                double* y = M + (size_t)prt * ld;
                double2 pv[NK];
#pragma unroll
                for (int k = 0; k < NK; ++k) pv[k] = *reinterpret_cast<const double2*>(y + c0 + 2 * LPP * k);
                const double ap = y[nslot];
                double g = 0.0, g1 = 0.0;
#pragma unroll
                for (int k = 0; k < NK; ++k) { g = fma(ov[k].x, pv[k].x, g);  g1 = fma(ov[k].y, pv[k].y, g1); }
                g += g1;
#pragma unroll
                for (int o = LPP / 2; o > 0; o >>= 1) g += __shfl_xor_sync(gmask, g, o);
                const double g2 = g * g, ab = ao * ap;
                if (ao > thr2 && ap > thr2 && g2 > rot2 * ab) {
                    big |= g2 > big2 * ab;
                    // d = |prt|^2 - |own|^2;  own' = cos own + so prt,  prt' = cos prt - so own with so = -sign(d) sin: the
                    // same rotation whichever member is held (the pair's Jacobi rotation does not depend on the order)
                    const double dd = ap - ao;
                    const double g24 = 4.0 * g2;
                    const double h2 = fma(dd, dd, g24);
                    const double u = fabs(dd) + h2 * fast_rsqrt1(h2);
                    const double w = fast_rsqrt1(fma(u, u, g24));
                    const double cs = u * w;
                    const double sn = 2.0 * g * w;
                    const bool own_grows = dd < 0.0;
                    const double so = own_grows ? sn : -sn;
                    // norms: the larger row grows by t g = 2 g^2 / u, the smaller shrinks by it
                    const double qn = 0.5 * g24 * fast_rcp(u);
                    const double apn = own_grows ? ap - qn : ap + qn;
                    ao = own_grows ? ao + qn : ao - qn;
                    if (t8 == 0) y[nslot] = apn;
#pragma unroll
                    for (int k = 0; k < NK; ++k) {
                        double2 on, pn;
                        on.x = fma(cs, ov[k].x, so * pv[k].x);  pn.x = fma(cs, pv[k].x, -so * ov[k].x);
                        on.y = fma(cs, ov[k].y, so * pv[k].y);  pn.y = fma(cs, pv[k].y, -so * ov[k].y);
                        ov[k] = on;
                        *reinterpret_cast<double2*>(y + c0 + 2 * LPP * k) = pn;
                    }
                }
                if (last) {     // the held row has met every other row: back to shared memory, adopt the next one
                    double* x = M + (size_t)own * ld;
#pragma unroll
                    for (int k = 0; k < NK; ++k) *reinterpret_cast<double2*>(x + c0 + 2 * LPP * k) = ov[k];
                    if (t8 == 0) x[nslot] = ao;
                    age = 0;
                    own += m;      if (own >= n1) own -= n1;
                    pm += m + 1;   if (pm >= n1) pm -= n1;
                } else {
                    ++age;
                    pm += 2;       if (pm >= n1) pm -= n1;
                }
            }
            __syncthreads();
            if (act && age == 0 && round + 1 < n1) {   // adopt: the row that was the minus member of pair n/2-1
#pragma unroll
                for (int k = 0; k < NK; ++k) ov[k] = *reinterpret_cast<const double2*>(M + (size_t)own * ld + c0 + 2 * LPP * k);
                ao = M[(size_t)own * ld + nslot];
            }
        }
        // end of sweep: every held row goes back (a group that has just released its row holds nothing new yet)
        if (act && age != 0) {
            double* x = M + (size_t)own * ld;
#pragma unroll
            for (int k = 0; k < NK; ++k) *reinterpret_cast<double2*>(x + c0 + 2 * LPP * k) = ov[k];
        }
        if (!__syncthreads_or(big)) { ++sweep; break; }
    }
    if (sweep >= 60 && threadIdx.x == 0) raise_flag(flags, FLAG_JACOBI_LIMIT);
    return sweep;
}

}  // namespace tnmc
