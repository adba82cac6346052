// tnmc_energy.cuh -- exact +-J energy (a-10, Eq. 1) and the independence
// Metropolis scan (a-11, Eq. 10).
#pragma once
#include <type_traits>

#include "tnmc_common.cuh"

namespace tnmc {

// E = -sum_<ij> J_ij s_i s_j on bit-packed rows.  For a bond with spins differing (x = 1) or not
// and coupling negative (n = 1) or not, J s s' = 1 - 2 (x ^ n); so with `nz` the mask of present
// bonds,  sum J s s' = popc(nz) - 2 popc((x ^ n) & nz).  One warp per configuration; lane l
// takes words l, l+32, ... of the (L x W)-word configuration, so loads are fully coalesced.
__global__ void energy_kernel(JView J, int L, int W, int dis_begin, int dis_count, int n_samples,
                              const uint32_t* __restrict__ cfg, int32_t* __restrict__ E) {
    const long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long n_cfg = (long long)dis_count * n_samples;
    if (wid >= n_cfg) return;
    const int lane = threadIdx.x & 31;
    const int dl = (int)(wid / n_samples);
    const int d = dis_begin + dl;
    const uint32_t* s = cfg + (size_t)wid * L * W;
    const uint32_t* rn = J.row(M_JR_NEG, d, 0);
    const uint32_t* rz = J.row(M_JR_NZ, d, 0);
    const uint32_t* dn = J.row(M_JD_NEG, d, 0);
    const uint32_t* dz = J.row(M_JD_NZ, d, 0);
    int acc = 0;
    const int n_words = L * W;
    for (int i = lane; i < n_words; i += 32) {
        const int w = i % W, r = i / W;
        const uint32_t cur = s[i];
        // right bonds: spin c against spin c+1 (bit 0 of the next word carries over)
        uint32_t nxt = cur >> 1;
        if (w + 1 < W) nxt |= s[i + 1] << 31;
        const uint32_t zr = rz[i];
        acc += __popc(zr) - 2 * __popc(((cur ^ nxt) ^ rn[i]) & zr);
        // down bonds: row r against row r+1
        if (r + 1 < L) {
            const uint32_t zd = dz[i];
            acc += __popc(zd) - 2 * __popc(((cur ^ s[i + W]) ^ dn[i]) & zd);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) E[wid] = -acc;
}

// Real-valued couplings (tnmc_create_real): E = -sum_<ij> J_ij s_i s_j in FP64.  One warp per configuration;
// lane l takes words l, l+32, ... and walks the 32 bonds of each word; the lane partial sums are combined in a
// fixed order, so the result is deterministic (it differs from another summation order by rounding only).
__global__ void energy_real_kernel(JView J, int L, int W, int dis_begin, int dis_count, int n_samples,
                                   const uint32_t* __restrict__ cfg, double* __restrict__ E) {
    const long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long n_cfg = (long long)dis_count * n_samples;
    if (wid >= n_cfg) return;
    const int lane = threadIdx.x & 31;
    const int d = dis_begin + (int)(wid / n_samples);
    const uint32_t* s = cfg + (size_t)wid * L * W;
    const double* jr = J.jr_real + (size_t)d * L * L;
    const double* jd = J.jd_real + (size_t)d * L * L;
    double acc = 0.0;
    for (int i = lane; i < L * W; i += 32) {
        const int w = i % W, r = i / W;
        const uint32_t cur = s[i];
        uint32_t nxt = cur >> 1;
        if (w + 1 < W) nxt |= s[i + 1] << 31;
        const uint32_t xr = cur ^ nxt;                                   // bit b: spins c and c+1 differ
        const uint32_t xd = r + 1 < L ? (cur ^ s[i + W]) : 0u;          // bit b: spins (r,c) and (r+1,c) differ
        const int nb = L - 32 * w < 32 ? L - 32 * w : 32;
        for (int b = 0; b < nb; ++b) {
            const int c = 32 * w + b;
            // bonds across the open boundary do not exist, whatever the caller stored there
            const double a = c + 1 < L ? jr[(size_t)r * L + c] : 0.0, bdn = r + 1 < L ? jd[(size_t)r * L + c] : 0.0;
            acc += ((xr >> b) & 1u) ? -a : a;
            acc += ((xd >> b) & 1u) ? -bdn : bdn;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) E[wid] = -acc;
}

// One thread per disorder: sequential scan over its proposals (readings G15/G16).  ET = int32 (+-J) or double.
template <typename ET>
__global__ void metropolis_kernel(double beta, int dis_begin, int dis_count, int n_samples,
                                  const ET* __restrict__ E, const double* __restrict__ logq,
                                  uint32_t seed_lo, uint32_t seed_hi, uint64_t step_offset,
                                  uint64_t first_disorder,
                                  double* cur_logq, ET* cur_E, int64_t* cur_idx,
                                  uint8_t* accepted, int64_t* n_accepted, double* sum_min1) {
    const int dl = blockIdx.x * blockDim.x + threadIdx.x;
    if (dl >= dis_count) return;
    const uint32_t ctr_dis = (uint32_t)(first_disorder + (uint64_t)(dis_begin + dl));
    double cq = cur_logq[dl];
    ET ce = cur_E[dl];
    long long ci = cur_idx[dl];
    long long nacc = 0;
    double smin = 0.0;
    const size_t base = (size_t)dl * n_samples;
    for (int n = 0; n < n_samples; ++n) {
        const ET en = E[base + n];
        const double qn = logq[base + n];
        const uint64_t stepi = step_offset + (uint64_t)n;
        if (ci < 0) {                 // empty chain: first proposal initialises it (not counted)
            ce = en; cq = qn; ci = (long long)stepi;
            accepted[base + n] = 1;
            continue;
        }
        const double logA = -beta * (double)(en - ce) + cq - qn;     // Eq. 10 in log form
        smin += logA < 0.0 ? exp(logA) : 1.0;
        const double u = philox_uniform(0u, (uint32_t)stepi, ctr_dis, TAG_METROPOLIS, seed_lo, seed_hi);
        const double logu = u > 0.0 ? log(u) : -INFINITY;
        if (logu < logA) {
            ce = en; cq = qn; ci = (long long)stepi;
            accepted[base + n] = 1;
            ++nacc;
        } else {
            accepted[base + n] = 0;
        }
    }
    cur_logq[dl] = cq; cur_E[dl] = ce; cur_idx[dl] = ci;
    n_accepted[dl] = nacc;
    if (sum_min1 != nullptr) sum_min1[dl] = smin;
}

// Magnetisation M = sum_i s_i of every configuration (popcount on the packed words): one warp per
// configuration, lanes stride over its L*W words.
__global__ void magnetisation_kernel(int L, int W, long long n_cfg, const uint32_t* __restrict__ cfg,
                                     int32_t* __restrict__ M) {
    const long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (wid >= n_cfg) return;
    const int lane = threadIdx.x & 31;
    const uint32_t* s = cfg + (size_t)wid * L * W;
    int up = 0;
    for (int i = lane; i < L * W; i += 32) up += __popc(s[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) up += __shfl_xor_sync(0xffffffffu, up, o);
    if (lane == 0) M[wid] = 2 * up - L * L;
}

// Thermal averages along the Metropolis chain (reading G19): at step n the chain sits on the last
// accepted proposal; every step adds E, E^2, M, |M|, M^2 of that state to the five accumulators.
// One thread per disorder, sequential over its proposals; exact integer arithmetic in 64 bits,
// added to the double accumulators once at the end.
template <typename ET>
__global__ void observables_kernel(int dis_count, int n_samples, const ET* __restrict__ E,
                                   const int32_t* __restrict__ M, const uint8_t* __restrict__ accepted,
                                   ET* cur_E, int32_t* cur_M, double* sums) {
    const int dl = blockIdx.x * blockDim.x + threadIdx.x;
    if (dl >= dis_count) return;
    // +-J: exact 64-bit integer sums; real couplings: FP64 sums in proposal order
    typedef typename std::conditional<std::is_same<ET, int32_t>::value, long long, double>::type AT;
    AT ce = cur_E[dl], s0 = 0, s1 = 0;
    long long cm = cur_M[dl], s2 = 0, s3 = 0, s4 = 0;
    const size_t base = (size_t)dl * n_samples;
    for (int n = 0; n < n_samples; ++n) {
        if (accepted[base + n]) { ce = E[base + n]; cm = M[base + n]; }
        s0 += ce; s1 += ce * ce; s2 += cm; s3 += cm < 0 ? -cm : cm; s4 += cm * cm;
    }
    cur_E[dl] = (ET)ce; cur_M[dl] = (int32_t)cm;
    double* o = sums + (size_t)dl * 5;
    o[0] += (double)s0; o[1] += (double)s1; o[2] += (double)s2; o[3] += (double)s3; o[4] += (double)s4;
}

// Replica overlap along two Metropolis chains of the same disorder (oracle/observables.replica_overlap): at step n
// chain x sits on its last accepted proposal at or before n (or on the carried state cur_x if none yet in this call);
// q_n = sum_i s_i^a s_i^b = N - 2 popc(a xor b) over the packed words (unused high bits are 0 in both).
// One warp per (disorder, step): the lanes find the two state indices by walking the flags backwards 32 at a time
// (ballot; the expected distance is 1 / p_acc), then stride over the L*W words.
__device__ __forceinline__ long long last_accepted_at_or_before(const uint8_t* __restrict__ acc, long long n, int lane) {
    for (long long hi = n; hi >= 0; hi -= 32) {
        const long long i = hi - lane;
        const unsigned m = __ballot_sync(0xffffffffu, i >= 0 && acc[i] != 0);
        if (m) return hi - (__ffs(m) - 1);
    }
    return -1;
}

__global__ void overlap_steps_kernel(int L, int W, int dis_count, int n_samples,
                                     const uint32_t* __restrict__ cfg_a, const uint8_t* __restrict__ acc_a,
                                     const uint32_t* __restrict__ cfg_b, const uint8_t* __restrict__ acc_b,
                                     const uint32_t* __restrict__ cur_a, const uint32_t* __restrict__ cur_b,
                                     int32_t* __restrict__ q_steps) {
    const long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (wid >= (long long)dis_count * n_samples) return;
    const int lane = threadIdx.x & 31;
    const int dl = (int)(wid / n_samples);
    const long long n = wid - (long long)dl * n_samples;
    const size_t base = (size_t)dl * n_samples, nw = (size_t)L * W;
    const long long ia = last_accepted_at_or_before(acc_a + base, n, lane);
    const long long ib = last_accepted_at_or_before(acc_b + base, n, lane);
    const uint32_t* a = ia >= 0 ? cfg_a + (base + (size_t)ia) * nw : cur_a + (size_t)dl * nw;
    const uint32_t* b = ib >= 0 ? cfg_b + (base + (size_t)ib) * nw : cur_b + (size_t)dl * nw;
    int diff = 0;
    for (int i = lane; i < (int)nw; i += 32) diff += __popc(a[i] ^ b[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
    if (lane == 0) q_steps[wid] = L * L - 2 * diff;
}

// One CTA per disorder: sums of q, |q|, q^2 over the steps of the call (exact 64-bit integers, added to the double
// accumulators once), then the chains' states leaving the call are copied into cur_a / cur_b.
__global__ void overlap_sums_kernel(int L, int W, int n_samples,
                                    const uint32_t* __restrict__ cfg_a, const uint8_t* __restrict__ acc_a,
                                    const uint32_t* __restrict__ cfg_b, const uint8_t* __restrict__ acc_b,
                                    const int32_t* __restrict__ q_steps, uint32_t* cur_a, uint32_t* cur_b, double* sums) {
    __shared__ long long red[3][32];
    __shared__ long long last[2];
    const int dl = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t base = (size_t)dl * n_samples, nw = (size_t)L * W;
    long long s0 = 0, s1 = 0, s2 = 0;
    for (int n = tid; n < n_samples; n += blockDim.x) {
        const long long q = q_steps[base + n];
        s0 += q; s1 += q < 0 ? -q : q; s2 += q * q;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, o);
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    if (lane == 0) { red[0][warp] = s0; red[1][warp] = s1; red[2][warp] = s2; }
    if (warp == 0) {
        const long long la = last_accepted_at_or_before(acc_a + base, n_samples - 1, lane);
        const long long lb = last_accepted_at_or_before(acc_b + base, n_samples - 1, lane);
        if (lane == 0) { last[0] = la; last[1] = lb; }
    }
    __syncthreads();
    if (tid == 0) {
        long long t0 = 0, t1 = 0, t2 = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { t0 += red[0][w]; t1 += red[1][w]; t2 += red[2][w]; }
        double* o = sums + (size_t)dl * 3;
        o[0] += (double)t0; o[1] += (double)t1; o[2] += (double)t2;
    }
    const long long la = last[0], lb = last[1];
    for (int i = tid; i < (int)nw; i += blockDim.x) {
        if (la >= 0) cur_a[(size_t)dl * nw + i] = cfg_a[(base + (size_t)la) * nw + i];
        if (lb >= 0) cur_b[(size_t)dl * nw + i] = cfg_b[(base + (size_t)lb) * nw + i];
    }
}

}  // namespace tnmc
