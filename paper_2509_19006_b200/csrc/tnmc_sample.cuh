// tnmc_sample.cuh -- row-by-row ancestral sampling (steps a-8, a-9 of DESIGN.md;
// SamplerIsing._sample_row).
//
// One CTA = one disorder x one tile of chains (samples); it walks all rows of its range with no
// inter-CTA dependency (chains never interact).  Per row: the right-environment
// sweep writes R_c to a CTA-private scratch in HBM, the left sweep
// reads it back.  Both sweeps are (chains x chi) x (chi x 2chi) products, run
// on the FP64 tensor pipe with mma.sync.m8n8k4.f64: 8 chains form the M dimension of one tile,
// the site tensor (shared by every chain of the disorder) is the B operand, staged through
// shared memory by a ring of TMA bulk copies (cp.async.bulk + mbarrier) that runs ahead across sweeps and rows.
//
// Fragment bookkeeping (see tnmc_common.cuh): with lane = 4*g + q,
//   A fragment (8x4):  lane holds  V[chain g][k-slot q]          of k-tile kt
//   B fragment (4x8):  lane holds  T[k-slot q][column g]         of (kt, nt)
//   C fragment (8x8):  lane holds  out[chain g][2q], [2q+1]      of n-tile nt
// and k-tile kt, slot q  <->  bond index 8*(kt/2) + 2q + (kt%2), so the C fragments of one site
// are, register for register, the A fragments of the next.
#pragma once
#include <type_traits>

#include "tnmc_common.cuh"

namespace tnmc {

constexpr int SAMPLE_WARPS = 8;
constexpr int SAMPLE_THREADS = SAMPLE_WARPS * 32;
constexpr int SAMPLE_MT = 2;                                   // 8-chain M tiles per warp
constexpr int SAMPLE_CHAINS = SAMPLE_WARPS * SAMPLE_MT * 8;    // chains per CTA
constexpr int SAMPLE_STAGES = 3;

struct SampleArgs {
    JView J;
    double beta;
    int L, chi;
    int dis_begin, n_samples;
    int row_lo, row_hi;              // rows [row_lo, row_hi)
    const int* slot_of_row;          // [L] device
    EnvRef env;                      // FP64 storage here; FP32 storage is read by tnmc_sample_tf32.cuh
    size_t env_dis_stride;           // elements per disorder
    double* renv;                    // scratch: per CTA  L * SAMPLE_CHAINS * P doubles
    uint32_t* cfg_bits;              // (dis_count, n_samples, L, W), or nullptr (tnmc_sample_fused: configurations not kept)
    int32_t* E_out;                  // (dis_count, n_samples) or nullptr: Eq. 1 accumulated in the left sweep (+-J only)
    int32_t* M_out;                  // (dis_count, n_samples) or nullptr: sum_i s_i, likewise
    uint32_t* carry;                 // (n_dis, n_samples_max, W): last row of a row range, for the next range when cfg_bits is nullptr
    int n_samples_max;
    const uint32_t* forced;          // or nullptr
    double* logq;                    // (dis_count, n_samples): accumulated over row ranges
    double* probs;                   // (dis_count, n_samples, L, L) or nullptr
    uint32_t seed_lo, seed_hi;
    uint64_t sample_offset, first_disorder;
    unsigned long long* flags;
};

__device__ __forceinline__ double quad_sum(double v) {
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    return v;
}

// MT_ = 8-chain M tiles per warp: 2 (128 chains per CTA, the default) or 1 (64 chains per CTA: twice the CTAs of half
// the size, chosen by the launcher when a 128-chain grid would leave SMs without work -- C2's 100 disorders x 100 samples)
template <int P, bool REALJ, bool F32READ, int MT_ = SAMPLE_MT>
__global__ void __launch_bounds__(SAMPLE_THREADS, MT_ == 1 ? 3 : 2) sample_rows_kernel(const SampleArgs args) {
    typedef typename std::conditional<F32READ, float, double>::type TS;   // storage type of the site tensors (TNMC_F32_STORE: float)
    constexpr int KT = P / 4;        // k tiles
    constexpr int NT = P / 4;        // n tiles (2P / 8)
    constexpr int JT = P / 8;        // 8-wide tiles per spin slice
    constexpr int MT = MT_;
    constexpr int CHAINS = SAMPLE_WARPS * MT * 8;      // chains per CTA
    constexpr int TSZ = 2 * P * P;
    extern __shared__ __align__(16) double smem[];
    double* sT = smem;                                                    // SAMPLE_STAGES * TSZ
    uint32_t* sBits = reinterpret_cast<uint32_t*>(smem + SAMPLE_STAGES * TSZ);  // [CHAINS][W] previous row

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, q = lane & 3;
    const int L = args.L, W = (L + 31) >> 5;
    // real couplings: (e^{beta J}, e^{-beta J}) of the up bonds of the current row, one entry per column
    double2* sJ = reinterpret_cast<double2*>(sBits + CHAINS * W);
    const int dl = blockIdx.y;                       // local disorder index (output indexing)
    const int d = args.dis_begin + dl;               // ctx disorder index (env / J indexing)
    const int tile = blockIdx.x;
    const double beta = args.beta;
    const double eb = exp(beta), emb = exp(-beta);
    const TS* env_d = reinterpret_cast<const TS*>(args.env.base) + (size_t)d * args.env_dis_stride;
    double* renv = args.renv + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * (size_t)L * CHAINS * P;

    // chain handled as M-tile mt, row g of this warp
    int chain_local[MT];      // index within the CTA
    long long samp[MT];       // sample index within this call (may be >= n_samples: inactive)
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        chain_local[mt] = (warp * MT + mt) * 8 + g;
        samp[mt] = (long long)tile * CHAINS + chain_local[mt];
    }
    // the "owner" lane of chain (mt = q, g) does that chain's scalar work
    const bool owner = q < MT;
    const int own_local = (warp * MT + (owner ? q : 0)) * 8 + g;
    const long long own_samp = (long long)tile * CHAINS + own_local;
    const bool own_active = owner && own_samp < args.n_samples;
    const size_t own_out = (size_t)dl * args.n_samples + (size_t)(own_active ? own_samp : 0);
    const uint32_t ctr_samp = (uint32_t)(args.sample_offset + (uint64_t)own_samp);
    const uint32_t ctr_dis = (uint32_t)(args.first_disorder + (uint64_t)d);

    double logq = 0.0;
    if (own_active && args.row_lo > 0) logq = args.logq[own_out];
    // fused energy / magnetisation (tnmc_sample_fused): the owner lane holds every finished word of the new row and
    // the word above it, which is all Eq. 1 needs: E = -sum J s s' by XOR + popcount, exactly as energy_kernel
    const bool fuse = !REALJ && args.E_out != nullptr;
    int eacc = 0, macc = 0;
    if (fuse && own_active && args.row_lo > 0) { eacc = args.E_out[own_out]; macc = args.M_out[own_out]; }
    uint32_t prev_w = 0, prev_rn = 0, prev_rz = 0;   // previous word of the row and its Jr masks (bond across the word boundary)

    // previous-row bits of this CTA's chains -> shared (zero for row 0: reading G9, no upper row)
    for (int t = tid; t < CHAINS * W; t += SAMPLE_THREADS) {
        const int cl = t / W, w = t % W;
        const long long s = (long long)tile * CHAINS + cl;
        uint32_t v = 0;
        if (args.row_lo > 0 && s < args.n_samples)
            v = args.cfg_bits != nullptr ? args.cfg_bits[(((size_t)dl * args.n_samples + s) * L + (args.row_lo - 1)) * W + w]
                                         : args.carry[((size_t)d * args.n_samples_max + s) * W + w];
        sBits[t] = v;
    }

    // ---- tensor stream: per row the right sweep consumes sites L-1..1, the left sweep sites 0..L-1
    const int steps_per_row = 2 * L - 1;
    const int n_rows = args.row_hi - args.row_lo;
    (void)n_rows;
    // the tensor stream is addressed with running counters (a 64-bit division per site costs ~60 instructions)
    int pf_r = args.row_lo, pf_t = 0, pf_stage = 0, cur_stage = 0;
    __shared__ uint64_t s_mbar[SAMPLE_STAGES];       // one mbarrier per stage of the tensor ring
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < SAMPLE_STAGES; ++s) mbar_init(&s_mbar[s], 1);
        mbar_init_fence();
    }
    __syncthreads();
    unsigned mbar_phase = 0;                          // bit s: parity of the next completion of stage s
    auto issue_prefetch = [&]() {
        if (pf_r < args.row_hi) {
            const int site = pf_t < L - 1 ? (L - 1 - pf_t) : (pf_t - (L - 1));
            const TS* src = env_d + ((size_t)args.slot_of_row[pf_r] * L + site) * TSZ;
            TS* dst = reinterpret_cast<TS*>(sT) + pf_stage * TSZ;
            if (tid == 0) {     // one bulk copy of the whole site tensor, completing on the stage's mbarrier
                mbar_expect_tx(&s_mbar[pf_stage], (unsigned)(TSZ * sizeof(TS)));
                bulk_copy_g2s(dst, src, (unsigned)(TSZ * sizeof(TS)), &s_mbar[pf_stage]);
            }
            if (++pf_t == steps_per_row) { pf_t = 0; ++pf_r; }
        }
        if (++pf_stage == SAMPLE_STAGES) pf_stage = 0;
    };
    for (int s = 0; s < SAMPLE_STAGES - 1; ++s) issue_prefetch();

    for (int r = args.row_lo; r < args.row_hi; ++r) {
        const bool has_up = r > 0;
        // ============================================================ right sweep
        double vf[MT][KT];          // current environment as A fragments
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) vf[mt][kt] = (kt == 0 && q == 0) ? 1.0 : 0.0;
        {   // R_{L-1} = [1]
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int jt = 0; jt < JT; ++jt) {
                    double2 v = make_double2((jt == 0 && q == 0) ? 1.0 : 0.0, 0.0);
                    double2* dst = reinterpret_cast<double2*>(
                        renv + ((((size_t)(L - 1) * SAMPLE_WARPS + warp) * MT + mt) * JT + jt) * 64) + lane;
                    *dst = v;
                }
        }
        if (REALJ) {
            __syncthreads();            // the previous row's left sweep is done with the table
            if (has_up)
                for (int c = tid; c < L; c += SAMPLE_THREADS) {
                    const double bj = args.beta * args.J.jd_real[((size_t)d * L + (r - 1)) * L + c];
                    sJ[c] = make_double2((double)exp(bj), (double)exp(-bj));
                }
        }
        uint32_t upw[MT];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) upw[mt] = 0u;
        uint32_t jneg = 0, jnz = 0;
        const uint32_t* jd_neg = has_up ? args.J.row(M_JD_NEG, d, r - 1) : nullptr;
        const uint32_t* jd_nz = has_up ? args.J.row(M_JD_NZ, d, r - 1) : nullptr;
        int cur_word = -1;
        for (int col = L - 2; col >= 0; --col) {
            mbar_wait(&s_mbar[cur_stage], (mbar_phase >> cur_stage) & 1u);   // the tensor of this step has landed
            mbar_phase ^= 1u << cur_stage;
            __syncthreads();            // everyone is done with the stage the next copy overwrites
            issue_prefetch();
            const TS* T = reinterpret_cast<const TS*>(sT) + cur_stage * TSZ;   // tensor of site col+1
            if (++cur_stage == SAMPLE_STAGES) cur_stage = 0;
            const int site = col + 1;
            if ((site >> 5) != cur_word) {
                cur_word = site >> 5;
                if (has_up) {
                    jneg = jd_neg[cur_word]; jnz = jd_nz[cur_word];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) upw[mt] = sBits[chain_local[mt] * W + cur_word];
                }
            }
            double acc[MT][NT][2];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) { acc[mt][nt][0] = 0.0; acc[mt][nt][1] = 0.0; }
            // out[chain][(a,i)] = sum_j T[i][a][j] R[chain][j]
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) {
                const int j = 8 * (kt >> 1) + 2 * q + (kt & 1);
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const int a = nt / JT, i = 8 * (nt % JT) + g;
                    const double b = (double)T[env_off(P, i, a, j)];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) dmma884(acc[mt][nt][0], acc[mt][nt][1], vf[mt][kt], b);
                }
            }
            // weights of the up bond for the two spin values
            const int bit = site & 31;
            const int jsign = has_up ? (((jnz >> bit) & 1u) ? (((jneg >> bit) & 1u) ? -1 : 1) : 0) : 0;
            // (e^{+beta J}, e^{-beta J}) of the up bond of this column: from the masks (+-J) or from the row table
            double ep, em;
            if (REALJ) { ep = has_up ? sJ[site].x : 1.0; em = has_up ? sJ[site].y : 1.0; }
            else { ep = jsign > 0 ? eb : (jsign < 0 ? emb : 1.0); em = jsign > 0 ? emb : (jsign < 0 ? eb : 1.0); }
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const bool up = (upw[mt] >> bit) & 1u;
                const double w1 = up ? ep : em, w0 = up ? em : ep;     // exp(+-beta J s_up) for the new spin up / down
                double nv[JT][2];
                double ss = 0.0;
#pragma unroll
                for (int it = 0; it < JT; ++it)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        nv[it][e] = w0 * acc[mt][it][e] + w1 * acc[mt][JT + it][e];
                        ss += nv[it][e] * nv[it][e];
                    }
                ss = quad_sum(ss);
                const double sc = ss > 0.0 ? rsqrt(ss) : 0.0;    // PAPER.md:238 (any positive scale is equivalent)
#pragma unroll
                for (int it = 0; it < JT; ++it) {
                    const double v0 = nv[it][0] * sc, v1 = nv[it][1] * sc;
                    vf[mt][2 * it] = v0;
                    vf[mt][2 * it + 1] = v1;
                    double2* dst = reinterpret_cast<double2*>(
                        renv + ((((size_t)col * SAMPLE_WARPS + warp) * MT + mt) * JT + it) * 64) + lane;
                    *dst = make_double2(v0, v1);
                }
            }
        }
        // ============================================================ left sweep
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int kt = 0; kt < KT; ++kt) vf[mt][kt] = (kt == 0 && q == 0) ? 1.0 : 0.0;
        cur_word = -1;
        uint32_t neww = 0;          // owner lane: bits of the current word of the new row
        uint32_t forcedw = 0;
        double prod = 1.0;          // owner lane: running product of chosen probabilities
        for (int col = 0; col < L; ++col) {
            mbar_wait(&s_mbar[cur_stage], (mbar_phase >> cur_stage) & 1u);   // the tensor of this step has landed
            mbar_phase ^= 1u << cur_stage;
            __syncthreads();            // everyone is done with the stage the next copy overwrites
            issue_prefetch();
            const TS* T = reinterpret_cast<const TS*>(sT) + cur_stage * TSZ;   // tensor of site col
            if (++cur_stage == SAMPLE_STAGES) cur_stage = 0;
            if ((col >> 5) != cur_word) {
                cur_word = col >> 5;
                if (has_up) {
                    jneg = jd_neg[cur_word]; jnz = jd_nz[cur_word];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) upw[mt] = sBits[chain_local[mt] * W + cur_word];
                }
                if (args.forced != nullptr && own_active)
                    forcedw = args.forced[(own_out * L + r) * W + cur_word];
                neww = 0;
            }
            double acc[MT][NT][2];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) { acc[mt][nt][0] = 0.0; acc[mt][nt][1] = 0.0; }
            // t[chain][(a,j)] = sum_i Lenv[chain][i] T[i][a][j]
#pragma unroll
            for (int kt = 0; kt < KT; ++kt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const double b = (double)T[(kt * NT + nt) * 32 + (lane ^ ((kt & 1) << 2))];
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) dmma884(acc[mt][nt][0], acc[mt][nt][1], vf[mt][kt], b);
                }
            // rho_a = | t_a . R_col |
            double rho0[MT], rho1[MT];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                double s0 = 0.0, s1 = 0.0;
#pragma unroll
                for (int jt = 0; jt < JT; ++jt) {
                    const double2 rv = *(reinterpret_cast<const double2*>(
                        renv + ((((size_t)col * SAMPLE_WARPS + warp) * MT + mt) * JT + jt) * 64) + lane);
                    s0 += acc[mt][jt][0] * rv.x + acc[mt][jt][1] * rv.y;
                    s1 += acc[mt][JT + jt][0] * rv.x + acc[mt][JT + jt][1] * rv.y;
                }
                rho0[mt] = fabs(quad_sum(s0));
                rho1[mt] = fabs(quad_sum(s1));
            }
            // owner lane: conditional probability (Eq. 5), draw, log q
            const int bit = col & 31;
            const int jsign = has_up ? (((jnz >> bit) & 1u) ? (((jneg >> bit) & 1u) ? -1 : 1) : 0) : 0;
            // (e^{+beta J}, e^{-beta J}) of the up bond of this column: from the masks (+-J) or from the row table
            double ep, em;
            if (REALJ) { ep = has_up ? sJ[col].x : 1.0; em = has_up ? sJ[col].y : 1.0; }
            else { ep = jsign > 0 ? eb : (jsign < 0 ? emb : 1.0); em = jsign > 0 ? emb : (jsign < 0 ? eb : 1.0); }
            int a_sel = 0;
            if (owner) {
                double r0 = rho0[0], r1 = rho1[0];
                uint32_t uw = upw[0];
#pragma unroll
                for (int mt = 1; mt < MT; ++mt) if (q == mt) { r0 = rho0[mt]; r1 = rho1[mt]; uw = upw[mt]; }
                if (r0 == 0.0 || r1 == 0.0) {          // reading G10: count and clamp
                    if (own_active) raise_flag(args.flags, FLAG_RHO_ZERO);
                    if (r0 == 0.0) r0 = 2.2250738585072014e-308;
                    if (r1 == 0.0) r1 = 2.2250738585072014e-308;
                }
                const bool up = (uw >> bit) & 1u;
                const double w1 = up ? ep : em, w0 = up ? em : ep;
                // sigma(log(r1/r0) + 2 beta J s_up) = r1 w1 / (r0 w0 + r1 w1)
                const double f0 = r0 * w0, f1 = r1 * w1;
                const double inv = 1.0 / (f0 + f1);
                const double p1 = f1 * inv, p0 = f0 * inv;
                const double u = philox_uniform((uint32_t)(r * L + col), ctr_samp, ctr_dis, TAG_SPIN,
                                                args.seed_lo, args.seed_hi);
                if (args.forced != nullptr) a_sel = (forcedw >> bit) & 1u;
                else a_sel = u < p1;
                if (own_active) {
                    if (!(p1 >= 0.0 && p1 <= 1.0)) raise_flag(args.flags, FLAG_NONFINITE);
                    if (fabs(u - p1) < 1e-9) raise_flag(args.flags, FLAG_NEAR_THRESHOLD);
                    if (args.probs != nullptr) args.probs[(own_out * L + r) * L + col] = p1;
                }
                prod *= a_sel ? p1 : p0;
                if (prod < 1e-200) { logq += log(prod); prod = 1.0; }
                neww |= (uint32_t)a_sel << bit;
                if (bit == 31 || col == L - 1) {
                    if (fuse) {
                        macc += 2 * __popc(neww) - (bit + 1);
                        // down bonds (r-1,c)-(r,c): (jneg, jnz) are the masks of Jd row r-1 for this word
                        if (has_up) eacc -= __popc(jnz) - 2 * __popc((uw ^ neww ^ jneg) & jnz);
                        // right bonds (r,c)-(r,c+1) inside the word; the bond out of bit 31 waits for the next word
                        const uint32_t rn = args.J.row(M_JR_NEG, d, r)[cur_word], rz = args.J.row(M_JR_NZ, d, r)[cur_word];
                        const uint32_t in = rz & 0x7fffffffu;
                        eacc -= __popc(in) - 2 * __popc(((neww ^ (neww >> 1)) ^ rn) & in);
                        if (cur_word > 0 && (prev_rz >> 31))
                            eacc -= 1 - 2 * (int)((((prev_w >> 31) ^ neww) ^ (prev_rn >> 31)) & 1u);
                        prev_w = neww; prev_rn = rn; prev_rz = rz;
                    }
                    if (own_active && args.cfg_bits != nullptr) args.cfg_bits[(own_out * L + r) * W + cur_word] = neww;
                    // sBits of this word is no longer needed by the left sweep: overwrite for the next row
                    sBits[own_local * W + cur_word] = neww;
                }
            }
            // environment update with the sampled slice
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const int sel = __shfl_sync(0xffffffffu, a_sel, (lane & ~3) | mt);
                double nv[JT][2];
                double ss = 0.0;
#pragma unroll
                for (int jt = 0; jt < JT; ++jt)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        nv[jt][e] = sel ? acc[mt][JT + jt][e] : acc[mt][jt][e];
                        ss += nv[jt][e] * nv[jt][e];
                    }
                ss = quad_sum(ss);
                const double sc = ss > 0.0 ? rsqrt(ss) : 0.0;
#pragma unroll
                for (int jt = 0; jt < JT; ++jt) {
                    vf[mt][2 * jt] = nv[jt][0] * sc;
                    vf[mt][2 * jt + 1] = nv[jt][1] * sc;
                }
            }
        }
        if (owner) { logq += log(prod); prod = 1.0; }
        __syncwarp();     // sBits written by owner lanes, read by the whole quad in the next row
    }
    if (own_active) args.logq[own_out] = logq;
    if (fuse && own_active) { args.E_out[own_out] = eacc; args.M_out[own_out] = macc; }
    if (args.cfg_bits == nullptr && args.row_hi < L) {     // configurations not kept: hand the last row to the next row range
        __syncthreads();
        for (int t = tid; t < CHAINS * W; t += SAMPLE_THREADS) {
            const long long s = (long long)tile * CHAINS + t / W;
            if (s < args.n_samples) args.carry[((size_t)d * args.n_samples_max + s) * W + t % W] = sBits[t];
        }
    }
}

}  // namespace tnmc
