// tnmc_common.cuh -- layouts, Philox4x32-10, fault counters shared by the CUDA kernels.
// (Part of the product path; shares nothing with oracle/.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace tnmc {

// ---------------------------------------------------------------------------------------------
// Fault counters (include/tnmc.h TNMC_FLAG_*)
// ---------------------------------------------------------------------------------------------
enum { FLAG_RHO_ZERO = 0, FLAG_NONFINITE = 1, FLAG_LOGZ_NONPOS = 2, FLAG_NEAR_THRESHOLD = 3,
       FLAG_JACOBI_LIMIT = 4, FLAG_SIGMA_ZERO = 5, N_FLAGS = 8 };

__device__ __forceinline__ void raise_flag(unsigned long long* flags, int which) {
    atomicAdd(flags + which, 1ull);
}

// ---------------------------------------------------------------------------------------------
// FP64 tensor-core primitive (DMMA in SASS; tcgen05 has no f64 kind, so mma.sync is the FP64 tensor path on sm_100a).
// With lane = 4 g + q:  A (8x4) lane holds A[g][q];  B (4x8) lane holds B[q][g];  C (8x8) lane holds C[g][2q], C[g][2q+1].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------------------------------------
// Bulk asynchronous copy global -> shared (TMA engine, `cp.async.bulk`, UBLKCP in SASS) completing on an mbarrier.
// A stored site tensor is one contiguous, 16-byte aligned block of 0.5 .. 16 KB: the ideal bulk copy -- one instruction by
// one thread per site instead of one 16-byte cp.async per thread and round.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                 :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "r"(bytes),
                    "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "TNMC_MBAR_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@p bra TNMC_MBAR_DONE;\n"
                 "bra TNMC_MBAR_WAIT;\n"
                 "TNMC_MBAR_DONE:\n"
                 "}" :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}

// One warp computes an 8-row strip of C = A B over NT 8-column tiles with DMMA: the A fragment of a k-step is loaded
// once and used for every column tile.  a_at(g, k), b_at(k, n) return the operand entries (0 outside the matrix),
// c_out(g, n, v) stores a result.  K is rounded up to a multiple of 4 by the callers' zero padding.
template <int NT, class FA, class FB, class FC>
__device__ __forceinline__ void dmma_strip(int K, int lane, FA a_at, FB b_at, FC c_out) {
    const int g = lane >> 2, q = lane & 3;
    double acc[NT][2];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) { acc[nt][0] = 0.0; acc[nt][1] = 0.0; }
#pragma unroll 4
    for (int k0 = 0; k0 < K; k0 += 4) {
        const double a = a_at(g, k0 + q);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) dmma884(acc[nt][0], acc[nt][1], a, b_at(k0 + q, 8 * nt + g));
    }
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) { c_out(g, 8 * nt + 2 * q, acc[nt][0]); c_out(g, 8 * nt + 2 * q + 1, acc[nt][1]); }
}

// ---------------------------------------------------------------------------------------------
// Environment site-tensor layout in HBM ("fragment order").
//
// A stored site tensor is A[i][a][j] (left bond i, spin a, right bond j), zero
// padded to P x 2 x P with P = 8, 16 or 32 (the smallest of these >= chi).  It is stored so that
// the left sampling sweep (contraction over i) can feed it to
// mma.sync.m8n8k4.f64 as the B operand with one conflict-free 8-byte shared-memory load per lane:
//   k-tile kt holds the four left-bond indices i = 8*(kt/2) + 2*q + (kt%2), q = 0..3
//   n-tile nt holds the eight columns (a, j) with a = nt / (P/8), j = 8*(nt % (P/8)) + g, g = 0..7
//   element offset = ((kt * NT + nt) * 32 + ((g*4 + q) ^ 4*(kt%2))),  NT = P/4,  lane = g*4 + q.
// The odd/even split of i over two k-tiles is what lets the accumulator fragment of one site
// (lane q holds columns 2q, 2q+1 of each n-tile) be used, unshuffled, as the A fragment of the
// next site.
// ---------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ int pad_chi(int chi) { return chi <= 8 ? 8 : (chi <= 16 ? 16 : 32); }

__host__ __device__ __forceinline__ int env_off(int P, int i, int a, int j) {
    const int kt = 2 * (i >> 3) + (i & 1);
    const int q = (i & 7) >> 1;
    const int nt = a * (P >> 3) + (j >> 3);
    const int g = j & 7;
    // odd k-tiles are stored with bit 2 of the in-tile index flipped: a permutation inside the tile for the left
    // sweep (still one conflict-free 8-byte load per lane), and it puts the two k-tile parities that the right
    // sweep's transposed read touches in one half-warp on disjoint banks
    return ((kt * (P >> 2) + nt) * 32 + ((g * 4 + q) ^ ((kt & 1) << 2)));
}

// FP32 storage (TNMC_F32_LOGSCALE) uses the fragment order of mma.sync.m16n8k8.tf32 instead: k-tile kt
// holds the eight left-bond indices i = 8*kt + 2*q + h (q = 0..3 <-> k-slots q and q+4 for h = 0, 1), the
// two values of a lane are adjacent and the even columns g of a tile come before the odd ones:
//   offset = ((kt * NT + nt) * 32 + (g&1)*16 + (g>>1)*4 + q) * 2 + h,  NT = P/4.
// The left sweep (contraction over i) reads its (b0, b1) pair with one conflict-free 8-byte load; the
// right sweep (contraction over j) reads the same tile transposed -- lane (g, q) needs
// (i = 8 it + g, j = 8 kt + 2q + e) -- at words 8q + g (e = 0) and 32 + 8q + g (e = 1): conflict-free too,
// which is what the even/odd split is for.  As in the FP64 layout the accumulator fragment of one site
// (columns 2q, 2q+1 of each n-tile) is the A fragment of the next.
__host__ __device__ __forceinline__ int env_off32(int P, int i, int a, int j) {
    const int kt = i >> 3;
    const int q = (i & 7) >> 1, h = i & 1;
    const int nt = a * (P >> 3) + (j >> 3);
    const int g = j & 7;
    return ((kt * (P >> 2) + nt) * 32 + (g & 1) * 16 + (g >> 1) * 4 + q) * 2 + h;
}
__host__ __device__ __forceinline__ int env_off_p(int P, int i, int a, int j, int f32) {
    return f32 ? env_off32(P, i, a, j) : env_off(P, i, a, j);
}

// The environment stack is stored in FP64 (TNMC_F64) or in FP32 (TNMC_F32_LOGSCALE: every stored row has
// unit 2-norm and carries its log-scale separately, so single precision has no range problem); offsets are
// in elements either way.
struct EnvRef {
    void* base;
    int f32;      // element type: float (TNMC_F32_LOGSCALE, TNMC_F32_STORE) or double
    int lay32;    // fragment order: env_off32 (TF32 sampler) or env_off (FP64 DMMA sampler)
    __device__ __forceinline__ double ld(size_t i) const {
        return f32 ? (double)reinterpret_cast<const float*>(base)[i] : reinterpret_cast<const double*>(base)[i];
    }
    __device__ __forceinline__ void st(size_t i, double v) const {
        if (f32) reinterpret_cast<float*>(base)[i] = (float)v; else reinterpret_cast<double*>(base)[i] = v;
    }
    __host__ __device__ __forceinline__ const char* bytes(size_t i) const {
        return reinterpret_cast<const char*>(base) + i * (f32 ? 4 : 8);
    }
};

// Bond dimension left of column c (c = 0..L) of the stored row r after compression (P-C2):
// min(chi, 2^min(c, L-c), 2^(L-r)); 1 at the two ends.  Closed form of the recurrences
//   q_{c+1} = min(2 q_c, D'_{c+1}),  k_c = min(chi, q_c, 2 k_{c+1})
// (checked against them by tests/test_host_logic.py).
__host__ __device__ __forceinline__ int row_bond(int L, int chi, int r, int c) {
    if (c <= 0 || c >= L) return 1;
    int e = c < L - c ? c : L - c;
    if (L - r < e) e = L - r;
    if (e >= 6) return chi;   // chi <= 32 < 2^6
    const int v = 1 << e;
    return v < chi ? v : chi;
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), restated from the published algorithm.
// Reading R of DESIGN.md: key = (seed lo, seed hi), counter = (site, sample, disorder, tag).
// ---------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2,
                                                      uint32_t& c3, uint32_t k0, uint32_t k1) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
}

// 53-bit uniform in [0,1) from the first two output words.
__host__ __device__ __forceinline__ double philox_uniform(uint32_t c0, uint32_t c1, uint32_t c2,
                                                          uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c0, c1, c2, c3, k0, k1);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    const uint64_t m = ((uint64_t)c0 << 21) | (uint64_t)(c1 >> 11);
    return (double)m * 1.1102230246251565e-16;  // 2^-53
}

enum { TAG_SPIN = 0, TAG_METROPOLIS = 1 };

// ---------------------------------------------------------------------------------------------
// Bit-packed couplings: for every disorder and row, W = ceil(L/32) words of each mask.
//   jr_neg bit c: Jr[r][c] < 0     jr_nz bit c: Jr[r][c] != 0
//   jd_neg bit c: Jd[r][c] < 0     jd_nz bit c: Jd[r][c] != 0
// stored as masks[(which * n_dis + d) * L * W + r * W + w], which = 0..3 in that order.
// ---------------------------------------------------------------------------------------------
enum { M_JR_NEG = 0, M_JR_NZ = 1, M_JD_NEG = 2, M_JD_NZ = 3 };

struct JView {
    const uint32_t* masks;
    const double* jr_real;   // (n_dis, L, L) real-valued couplings (tnmc_create_real), else nullptr
    const double* jd_real;
    int n_dis, L, W;
    // coupling value as a double: the real array if there is one, else the +-1 / 0 of the masks
    __device__ __forceinline__ double jrv(int d, int r, int c) const {
        return jr_real ? jr_real[((size_t)d * L + r) * L + c] : (double)jr(d, r, c);
    }
    __device__ __forceinline__ double jdv(int d, int r, int c) const {
        return jd_real ? jd_real[((size_t)d * L + r) * L + c] : (double)jd(d, r, c);
    }
    __device__ __forceinline__ const uint32_t* row(int which, int d, int r) const {
        return masks + ((size_t)which * n_dis + d) * (size_t)L * W + (size_t)r * W;
    }
    // coupling value in {-1,0,+1}
    __device__ __forceinline__ int jr(int d, int r, int c) const {
        const uint32_t nz = row(M_JR_NZ, d, r)[c >> 5] >> (c & 31) & 1u;
        const uint32_t ng = row(M_JR_NEG, d, r)[c >> 5] >> (c & 31) & 1u;
        return nz ? (ng ? -1 : 1) : 0;
    }
    __device__ __forceinline__ int jd(int d, int r, int c) const {
        const uint32_t nz = row(M_JD_NZ, d, r)[c >> 5] >> (c & 31) & 1u;
        const uint32_t ng = row(M_JD_NEG, d, r)[c >> 5] >> (c & 31) & 1u;
        return nz ? (ng ? -1 : 1) : 0;
    }
};

}  // namespace tnmc
