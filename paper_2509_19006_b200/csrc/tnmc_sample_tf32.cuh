// tnmc_sample_tf32.cuh -- the sampler of the reduced-precision mode TNMC_F32_LOGSCALE (steps a-8, a-9;
// SamplerIsing._sample_row; the paper's own dtype is torch.float).
//
// Same structure as tnmc_sample.cuh (one CTA = one disorder x 128 chains, walks all rows; right sweep
// writes the right environments to a CTA-private scratch, left sweep reads them back), with
//   * site tensors stored in FP32 (half the stack) in the fragment order of mma.sync.m16n8k8.tf32
//     (env_off32, tnmc_common.cuh), streamed by the same cp.async ring and fed to the tensor cores as
//     raw FP32 words (the hardware reads the TF32 subset: 10 mantissa bits), FP32 accumulation;
//   * 16 chains form the M dimension of a tile: rows g and g+8 of the fragment are two chains, which
//     play the role of the two M tiles of the FP64 kernel, so chain numbering and ownership are identical;
//   * environments normalised per site in FP32 -- that per-site normalisation is
//     the log-scaling that keeps single precision in range;
//   * the conditional probability, the draw and log q in FP64 from the FP32 weights rho_a: p0 = 1 - p1
//     exactly and log q is the log of the probabilities the draw used, so q is a normalised distribution
//     and the Metropolis correction (Eq. 10) stays exact whatever the rounding of the contractions.
#pragma once
#include "tnmc_linalg.cuh"
#include "tnmc_sample.cuh"

namespace tnmc {

__device__ __forceinline__ void mma16808_tf32(float& c0, float& c1, float& c2, float& c3,
                                              float a0, float a1, float a2, float a3, float b0, float b1) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(c0), "+f"(c1), "+f"(c2), "+f"(c3)
                 : "r"(__float_as_uint(a0)), "r"(__float_as_uint(a1)), "r"(__float_as_uint(a2)), "r"(__float_as_uint(a3)),
                   "r"(__float_as_uint(b0)), "r"(__float_as_uint(b1)));
}

// Error-compensated product (3xTF32): x = hi + lo with hi the TF32 part (top 19 bits) and lo = x - hi exact in
// FP32; a b ~ a_lo b_hi + a_hi b_lo + a_hi b_hi (small terms first), three MMAs, FP32-level accuracy (~1e-6)
// instead of TF32's ~5e-4 per product.
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

template <bool X3>
__device__ __forceinline__ void mma_tf32_x(float& c0, float& c1, float& c2, float& c3,
                                           float a0, float a1, float a2, float a3, float b0, float b1) {
    if (X3) {
        const float a0h = tf32_hi(a0), a1h = tf32_hi(a1), a2h = tf32_hi(a2), a3h = tf32_hi(a3);
        const float b0h = tf32_hi(b0), b1h = tf32_hi(b1);
        mma16808_tf32(c0, c1, c2, c3, a0 - a0h, a1 - a1h, a2 - a2h, a3 - a3h, b0h, b1h);
        mma16808_tf32(c0, c1, c2, c3, a0h, a1h, a2h, a3h, b0 - b0h, b1 - b1h);
        mma16808_tf32(c0, c1, c2, c3, a0h, a1h, a2h, a3h, b0h, b1h);
    } else {
        mma16808_tf32(c0, c1, c2, c3, a0, a1, a2, a3, b0, b1);
    }
}

__device__ __forceinline__ float quad_sumf(float v) {
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    return v;
}

template <int P, bool REALJ, bool X3>
__global__ void __launch_bounds__(SAMPLE_THREADS, X3 ? 3 : 2) sample_rows_tf32_kernel(const SampleArgs args) {
    constexpr int KT8 = P / 8;       // k tiles (8 bond indices each)
    constexpr int NT = P / 4;        // n tiles (2P / 8)
    constexpr int JT = P / 8;        // 8-wide tiles per spin slice
    constexpr int MT = SAMPLE_MT;    // the two 8-chain halves (rows g, g + 8) of the 16-row M tile
    constexpr int TSZ = 2 * P * P;
    static_assert(SAMPLE_MT == 2, "rows g and g+8 of the m16 fragment stand for the two M tiles");
    extern __shared__ __align__(16) float smem_f[];
    float* sT = smem_f;                                                            // SAMPLE_STAGES * TSZ
    uint32_t* sBits = reinterpret_cast<uint32_t*>(smem_f + SAMPLE_STAGES * TSZ);   // [SAMPLE_CHAINS][W] previous row

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, q = lane & 3;
    const int L = args.L, W = (L + 31) >> 5;
    // real couplings: (e^{beta J}, e^{-beta J}) of the up bonds of the current row, one entry per column
    float2* sJ = reinterpret_cast<float2*>(sBits + SAMPLE_CHAINS * W);
    const int dl = blockIdx.y;
    const int d = args.dis_begin + dl;
    const int tile = blockIdx.x;
    const float beta = (float)args.beta;
    const float eb = expf(beta), emb = expf(-beta);
    const size_t env_d = (size_t)d * args.env_dis_stride;
    float* renv = reinterpret_cast<float*>(args.renv + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * (size_t)L * SAMPLE_CHAINS * P);

    int chain_local[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) chain_local[mt] = (warp * MT + mt) * 8 + g;
    const bool owner = q < MT;
    const int own_local = (warp * MT + (owner ? q : 0)) * 8 + g;
    const long long own_samp = (long long)tile * SAMPLE_CHAINS + own_local;
    const bool own_active = owner && own_samp < args.n_samples;
    const size_t own_out = (size_t)dl * args.n_samples + (size_t)(own_active ? own_samp : 0);
    const uint32_t ctr_samp = (uint32_t)(args.sample_offset + (uint64_t)own_samp);
    const uint32_t ctr_dis = (uint32_t)(args.first_disorder + (uint64_t)d);

    double logq = 0.0;
    if (own_active && args.row_lo > 0) logq = args.logq[own_out];
    // fused energy / magnetisation (tnmc_sample_fused), as in sample_rows_kernel
    const bool fuse = !REALJ && args.E_out != nullptr;
    int eacc = 0, macc = 0;
    if (fuse && own_active && args.row_lo > 0) { eacc = args.E_out[own_out]; macc = args.M_out[own_out]; }
    uint32_t prev_w = 0, prev_rn = 0, prev_rz = 0;

    for (int t = tid; t < SAMPLE_CHAINS * W; t += SAMPLE_THREADS) {
        const int cl = t / W, w = t % W;
        const long long s = (long long)tile * SAMPLE_CHAINS + cl;
        uint32_t v = 0;
        if (args.row_lo > 0 && s < args.n_samples)
            v = args.cfg_bits != nullptr ? args.cfg_bits[(((size_t)dl * args.n_samples + s) * L + (args.row_lo - 1)) * W + w]
                                         : args.carry[((size_t)d * args.n_samples_max + s) * W + w];
        sBits[t] = v;
    }

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
            const float* src = reinterpret_cast<const float*>(args.env.base) + env_d + ((size_t)args.slot_of_row[pf_r] * L + site) * TSZ;
            float* dst = sT + pf_stage * TSZ;
            if (tid == 0) {     // one bulk copy of the whole site tensor, completing on the stage's mbarrier
                mbar_expect_tx(&s_mbar[pf_stage], (unsigned)(TSZ * sizeof(float)));
                bulk_copy_g2s(dst, src, (unsigned)(TSZ * sizeof(float)), &s_mbar[pf_stage]);
            }
            if (++pf_t == steps_per_row) { pf_t = 0; ++pf_r; }
        }
        if (++pf_stage == SAMPLE_STAGES) pf_stage = 0;
    };
    for (int s = 0; s < SAMPLE_STAGES - 1; ++s) issue_prefetch();

    for (int r = args.row_lo; r < args.row_hi; ++r) {
        const bool has_up = r > 0;
        // ============================================================ right sweep
        float vf[MT][2 * KT8];      // current environment: A fragments (a0,a2) of chain half 0, (a1,a3) of half 1
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int k = 0; k < 2 * KT8; ++k) vf[mt][k] = (k == 0 && q == 0) ? 1.0f : 0.0f;
        {   // R_{L-1} = [1]
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int jt = 0; jt < JT; ++jt) {
                    float2* dst = reinterpret_cast<float2*>(
                        renv + ((((size_t)(L - 1) * SAMPLE_WARPS + warp) * MT + mt) * JT + jt) * 64) + lane;
                    *dst = make_float2((jt == 0 && q == 0) ? 1.0f : 0.0f, 0.0f);
                }
        }
        if (REALJ) {
            __syncthreads();            // the previous row's left sweep is done with the table
            if (has_up)
                for (int c = tid; c < L; c += SAMPLE_THREADS) {
                    const double bj = args.beta * args.J.jd_real[((size_t)d * L + (r - 1)) * L + c];
                    sJ[c] = make_float2((float)exp(bj), (float)exp(-bj));
                }
        }
        uint32_t upw[MT] = {0u, 0u};
        uint32_t jneg = 0, jnz = 0;
        const uint32_t* jd_neg = has_up ? args.J.row(M_JD_NEG, d, r - 1) : nullptr;
        const uint32_t* jd_nz = has_up ? args.J.row(M_JD_NZ, d, r - 1) : nullptr;
        int cur_word = -1;
        for (int col = L - 2; col >= 0; --col) {
            mbar_wait(&s_mbar[cur_stage], (mbar_phase >> cur_stage) & 1u);   // the tensor of this step has landed
            mbar_phase ^= 1u << cur_stage;
            __syncthreads();            // everyone is done with the stage the next copy overwrites
            issue_prefetch();
            const float* T = sT + cur_stage * TSZ;   // tensor of site col+1
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
            float acc[MT][NT][2];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) { acc[mt][nt][0] = 0.0f; acc[mt][nt][1] = 0.0f; }
            // out[chain][(a,i)] = sum_j T[i][a][j] R[chain][j]:  k-slots q, q+4 of k-tile kt <-> j = 8 kt + 2q, 8 kt + 2q + 1
#pragma unroll
            for (int kt = 0; kt < KT8; ++kt) {
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const int a = nt / JT, it = nt % JT;
                    const int off = (it * NT + a * JT + kt) * 64 + 8 * q + g;   // env_off32(P, 8 it + g, a, 8 kt + 2q); the odd column is 32 words on
                    const float b0 = T[off], b1 = T[off + 32];
                    mma_tf32_x<X3>(acc[0][nt][0], acc[0][nt][1], acc[1][nt][0], acc[1][nt][1],
                                  vf[0][2 * kt], vf[1][2 * kt], vf[0][2 * kt + 1], vf[1][2 * kt + 1], b0, b1);
                }
            }
            // weights of the up bond for the two spin values
            const int bit = site & 31;
            const int jsign = has_up ? (((jnz >> bit) & 1u) ? (((jneg >> bit) & 1u) ? -1 : 1) : 0) : 0;
            // (e^{+beta J}, e^{-beta J}) of the up bond of this column: from the masks (+-J) or from the row table
            float ep, em;
            if (REALJ) { ep = has_up ? sJ[site].x : 1.0f; em = has_up ? sJ[site].y : 1.0f; }
            else { ep = jsign > 0 ? eb : (jsign < 0 ? emb : 1.0f); em = jsign > 0 ? emb : (jsign < 0 ? eb : 1.0f); }
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const bool up = (upw[mt] >> bit) & 1u;
                const float w1 = up ? ep : em, w0 = up ? em : ep;     // exp(+-beta J s_up) for the new spin up / down
                float nv[JT][2];
                float ss = 0.0f;
#pragma unroll
                for (int it = 0; it < JT; ++it)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        nv[it][e] = w0 * acc[mt][it][e] + w1 * acc[mt][JT + it][e];
                        ss += nv[it][e] * nv[it][e];
                    }
                ss = quad_sumf(ss);
                const float sc = ss > 0.0f ? rsqrtf(ss) : 0.0f;    // PAPER.md:238 (any positive scale is equivalent)
#pragma unroll
                for (int it = 0; it < JT; ++it) {
                    const float v0 = nv[it][0] * sc, v1 = nv[it][1] * sc;
                    vf[mt][2 * it] = v0;
                    vf[mt][2 * it + 1] = v1;
                    float2* dst = reinterpret_cast<float2*>(
                        renv + ((((size_t)col * SAMPLE_WARPS + warp) * MT + mt) * JT + it) * 64) + lane;
                    *dst = make_float2(v0, v1);
                }
            }
        }
        // ============================================================ left sweep
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int k = 0; k < 2 * KT8; ++k) vf[mt][k] = (k == 0 && q == 0) ? 1.0f : 0.0f;
        cur_word = -1;
        uint32_t neww = 0;          // owner lane: bits of the current word of the new row
        uint32_t forcedw = 0;
        double prod = 1.0;          // owner lane: running product of chosen probabilities
        for (int col = 0; col < L; ++col) {
            mbar_wait(&s_mbar[cur_stage], (mbar_phase >> cur_stage) & 1u);   // the tensor of this step has landed
            mbar_phase ^= 1u << cur_stage;
            __syncthreads();            // everyone is done with the stage the next copy overwrites
            issue_prefetch();
            const float* T = sT + cur_stage * TSZ;   // tensor of site col
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
            // right environments of this column: loaded before the MMAs so that their latency is covered
            float2 rv[MT][JT];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int jt = 0; jt < JT; ++jt)
                    rv[mt][jt] = *(reinterpret_cast<const float2*>(
                        renv + ((((size_t)col * SAMPLE_WARPS + warp) * MT + mt) * JT + jt) * 64) + lane);
            float acc[MT][NT][2];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) { acc[mt][nt][0] = 0.0f; acc[mt][nt][1] = 0.0f; }
            // t[chain][(a,j)] = sum_i Lenv[chain][i] T[i][a][j]
#pragma unroll
            for (int kt = 0; kt < KT8; ++kt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const float2 b = *(reinterpret_cast<const float2*>(T) + (kt * NT + nt) * 32 + (g & 1) * 16 + (g >> 1) * 4 + q);
                    mma_tf32_x<X3>(acc[0][nt][0], acc[0][nt][1], acc[1][nt][0], acc[1][nt][1],
                                  vf[0][2 * kt], vf[1][2 * kt], vf[0][2 * kt + 1], vf[1][2 * kt + 1], b.x, b.y);
                }
            // rho_a = | t_a . R_col |
            float rho0[MT], rho1[MT];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                float s0 = 0.0f, s1 = 0.0f;
#pragma unroll
                for (int jt = 0; jt < JT; ++jt) {
                    s0 += acc[mt][jt][0] * rv[mt][jt].x + acc[mt][jt][1] * rv[mt][jt].y;
                    s1 += acc[mt][JT + jt][0] * rv[mt][jt].x + acc[mt][JT + jt][1] * rv[mt][jt].y;
                }
                rho0[mt] = fabsf(quad_sumf(s0));
                rho1[mt] = fabsf(quad_sumf(s1));
            }
            // owner lane: conditional probability (Eq. 5), draw, log q -- in FP64
            const int bit = col & 31;
            const int jsign = has_up ? (((jnz >> bit) & 1u) ? (((jneg >> bit) & 1u) ? -1 : 1) : 0) : 0;
            // (e^{+beta J}, e^{-beta J}) of the up bond of this column: from the masks (+-J) or from the row table
            float ep, em;
            if (REALJ) { ep = has_up ? sJ[col].x : 1.0f; em = has_up ? sJ[col].y : 1.0f; }
            else { ep = jsign > 0 ? eb : (jsign < 0 ? emb : 1.0f); em = jsign > 0 ? emb : (jsign < 0 ? eb : 1.0f); }
            int a_sel = 0;
            if (owner) {
                float r0 = rho0[0], r1 = rho1[0];
                uint32_t uw = upw[0];
#pragma unroll
                for (int mt = 1; mt < MT; ++mt) if (q == mt) { r0 = rho0[mt]; r1 = rho1[mt]; uw = upw[mt]; }
                if (r0 == 0.0f || r1 == 0.0f) {        // reading G10: count and clamp (to the smallest normal FP32)
                    if (own_active) raise_flag(args.flags, FLAG_RHO_ZERO);
                    if (r0 == 0.0f) r0 = 1.1754943508222875e-38f;
                    if (r1 == 0.0f) r1 = 1.1754943508222875e-38f;
                }
                const bool up = (uw >> bit) & 1u;
                const float w1 = up ? ep : em, w0 = up ? em : ep;
                // sigma(log(r1/r0) + 2 beta J s_up) = r1 w1 / (r0 w0 + r1 w1) in FP32 (r's scaled against overflow of
                // the sum: both are <= 1 by the normalisation); p1 is then a fixed FP64 number and p0 = 1 - p1 exactly
                const float f0 = r0 * w0, f1 = r1 * w1;
                const double p1 = (double)fminf(__fdividef(f1, f0 + f1), 1.0f), p0 = 1.0 - p1;
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
                        if (has_up) eacc -= __popc(jnz) - 2 * __popc((uw ^ neww ^ jneg) & jnz);
                        const uint32_t rn = args.J.row(M_JR_NEG, d, r)[cur_word], rz = args.J.row(M_JR_NZ, d, r)[cur_word];
                        const uint32_t in = rz & 0x7fffffffu;
                        eacc -= __popc(in) - 2 * __popc(((neww ^ (neww >> 1)) ^ rn) & in);
                        if (cur_word > 0 && (prev_rz >> 31))
                            eacc -= 1 - 2 * (int)((((prev_w >> 31) ^ neww) ^ (prev_rn >> 31)) & 1u);
                        prev_w = neww; prev_rn = rn; prev_rz = rz;
                    }
                    if (own_active && args.cfg_bits != nullptr) args.cfg_bits[(own_out * L + r) * W + cur_word] = neww;
                    sBits[own_local * W + cur_word] = neww;
                }
            }
            // environment update with the sampled slice
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const int sel = __shfl_sync(0xffffffffu, a_sel, (lane & ~3) | mt);
                float nv[JT][2];
                float ss = 0.0f;
#pragma unroll
                for (int jt = 0; jt < JT; ++jt)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        nv[jt][e] = sel ? acc[mt][JT + jt][e] : acc[mt][jt][e];
                        ss += nv[jt][e] * nv[jt][e];
                    }
                ss = quad_sumf(ss);
                const float sc = ss > 0.0f ? rsqrtf(ss) : 0.0f;
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
        for (int t = tid; t < SAMPLE_CHAINS * W; t += SAMPLE_THREADS) {
            const long long s = (long long)tile * SAMPLE_CHAINS + t / W;
            if (s < args.n_samples) args.carry[((size_t)d * args.n_samples_max + s) * W + t % W] = sBits[t];
        }
    }
}

}  // namespace tnmc
