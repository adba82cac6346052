/* tnmc.h -- C ABI of the B200-native BatchTNMC hot path (arXiv 2509.19006).
 *
 * Citations "PAPER.md:NN" refer to /root/reference/PAPER.md; "DESIGN.md Gn / P-C2 / R" are the
 * readings of the paper listed in DESIGN.md.
 *
 * What the library computes, per disorder realisation d of the 2D +-J Ising model on an open
 * L x L lattice (Eq. 1):
 *   tnmc_build_envs  the boundary-MPS "cache" of create_cache_ising: the row
 *                    MPOs of Eq. 7-8 applied bottom-to-top to the
 *                    bottom-row MPS, each product compressed to bond
 *                    dimension chi (multiply/compress, PAPER.md:97 Fig. 2, :147, :186-187;
 *                    reading P-C2), and log Z (Eq. 6);
 *   tnmc_sample      SamplerIsing.sample/_sample_row: row-by-row ancestral
 *                    sampling with the right-environment sweep and the left
 *                    sampling sweep (Eq. 5), returning bit-packed
 *                    configurations and log q(s) (Eq. 9);
 *   tnmc_energy      Eq. 1, exact integer arithmetic;
 *   tnmc_metropolis  the independence Metropolis-Hastings acceptance of Eq. 10;
 *   tnmc_observables thermal averages of E and M along the accepted chain.
 *
 * Conventions
 *   rows r = 0..L-1 top to bottom, columns c = 0..L-1 left to right, raster order
 *   site = r*L + c; spin index a in {0,1} <-> s = 2a-1.
 *   Jr[d][r][c] couples (r,c)-(r,c+1) (the paper's J_mat[r,c,2]), must be 0 at
 *   c = L-1; Jd[d][r][c] couples (r,c)-(r+1,c) (J_mat[r,c,3]), must be 0 at r = L-1.
 *   cfg_bits: uint32 (dis_count, n_samples, L, W) with W = ceil(L/32); bit (c % 32) of word
 *   c/32 of row r is 1 iff s(r,c) = +1; unused high bits are 0.
 *   Random numbers (reading R): Philox4x32-10, key = (seed & 0xffffffff, seed >> 32),
 *   counter = (site, sample index, disorder index, tag), tag 0 = spin draws, tag 1 = Metropolis
 *   draws (site word 0, sample word = step index); u = ((x0 << 21) | (x1 >> 11)) * 2^-53;
 *   a spin is +1 iff u < p.  "disorder index" is first_disorder + d, "sample index" is
 *   sample_offset + n, so results do not depend on how calls are chunked.  Each of the three indices fills ONE
 *   32-bit counter word: first_disorder + n_dis, sample_offset + n_samples and step_offset + n_samples must not
 *   exceed 2^32 (TNMC_EINVAL otherwise) -- the configs of the paper use at most 10^3 of each.
 *
 * Memory and ownership
 *   Every pointer marked [dev] is a device pointer owned by the caller (e.g. torch tensors);
 *   [host] is a host pointer.  The context owns only a few hundred bytes of host metadata; all
 *   device storage it uses lives inside the caller-provided workspace (size from
 *   tnmc_workspace_bytes), which must stay alive and untouched until tnmc_destroy.  No entry
 *   point allocates device memory.  Kernels are enqueued on the stream given to tnmc_create and
 *   the calls return before completion; outputs are valid after the caller synchronises that
 *   stream.  Only tnmc_get_flags / tnmc_get_env_row / tnmc_run_host synchronise (tnmc_create does not: its slot
 *   maps and coupling masks are written by kernels on the stream).
 *
 * Errors
 *   Every call returns a tnmc_status; nothing throws across the ABI.  Argument errors are
 *   detected synchronously and leave the context unchanged; tnmc_last_error gives a message.
 *   Numeric faults inside kernels (rho == 0, non-finite values, non-positive sum for log Z,
 *   Jacobi sweep limit) are counted on the device and read with tnmc_get_flags.
 *   There is no CPU fallback anywhere: without a CUDA device every compute call fails with
 *   TNMC_ECUDA.
 */
#ifndef TNMC_H_
#define TNMC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tnmc_ctx tnmc_ctx; /* opaque, library-owned host object */

typedef enum {
    TNMC_OK = 0,
    TNMC_EINVAL = 1,   /* bad argument */
    TNMC_ENOMEM = 2,   /* workspace too small */
    TNMC_ECUDA = 3,    /* CUDA runtime error (message in tnmc_last_error) */
    TNMC_ESTATE = 4,   /* call order: e.g. tnmc_sample before tnmc_build_envs */
    TNMC_ENUMERIC = 5
} tnmc_status;

typedef enum {
    TNMC_F64 = 0,          /* FP64 storage and arithmetic: the parity path (log Z 1e-10, conditionals 1e-9) */
    TNMC_F32_LOGSCALE = 1, /* reduced precision (BASELINE configs[2]; the paper's own dtype is torch.float):
                              environment stack stored in FP32 -- every stored row has unit 2-norm and carries
                              its log-scale separately (reading G7), so single precision has no range problem --
                              and sampling contractions on TF32 tensor cores (mma.sync.m16n8k8, FP32 accumulate,
                              environments normalised per site) with 3xTF32 error compensation (each operand
                              split into its TF32 part and the exact FP32 remainder, three MMAs per product):
                              FP32-level accuracy, ~1e-6 per conditional.  The compression stays FP64 (it has to resolve
                              sigma_chi / sigma_1 ~ 1e-9).  Conditional probabilities, the draw and log q are
                              evaluated in FP64 from the FP32 weights with p0 = 1 - p1: q is a normalised
                              distribution and log q is the log of the probabilities actually used, so the
                              Metropolis correction stays exact.  log Z agrees with TNMC_F64 to ~1e-7 relative
                              (north_star reduced-precision tolerance 1e-4); spins are not bit-identical to the
                              FP64 path.
                              TNMC_FLAG_RHO_ZERO is informational in this mode. */
    TNMC_F32_STORE = 2,    /* environment stack stored in FP32 (in the FP64 sampler's fragment order), ALL arithmetic
                              FP64: the tensors are rounded to FP32 once when a row is stored, the compression and
                              the FP64 DMMA sampler read them back as doubles.  Half the HBM footprint and stack
                              traffic at conditionals within ~1e-6 of TNMC_F64 and an unchanged acceptance; spins
                              are not bit-identical to TNMC_F64.  q is normalised and log q is the log of the
                              probabilities used, as in every mode. */
    TNMC_TF32_FAST = 3     /* as TNMC_F32_LOGSCALE with plain TF32 products (one MMA, 10-bit mantissa inputs): the
                              fastest sampler (HBM-bound), ~1e-3 of noise per conditional, noticeably lower
                              acceptance on large lattices.  q stays normalised and log q consistent. */
} tnmc_prec;

/* indices into the array returned by tnmc_get_flags */
enum {
    TNMC_FLAG_RHO_ZERO = 0,      /* a conditional weight rho_a was exactly 0 (reading G10) */
    TNMC_FLAG_NONFINITE = 1,     /* a non-finite intermediate was seen */
    TNMC_FLAG_LOGZ_NONPOS = 2,   /* sum_sigma Psi_0(sigma) <= 0 in the log Z read-out */
    TNMC_FLAG_NEAR_THRESHOLD = 3,/* draws with |u - p| < 1e-9 (north_star parity clause) */
    TNMC_FLAG_JACOBI_LIMIT = 4,  /* a site SVD hit the sweep limit before converging */
    TNMC_FLAG_SIGMA_ZERO = 5,    /* informational: a kept singular value was below the numerical rank (exact-chi cases) */
    TNMC_N_FLAGS = 8
};

/* Size in bytes of the workspace tnmc_create needs.
 *   L >= 2, 2 <= chi <= 32, n_dis >= 1, n_samples_max >= 1 (largest n_samples of any later
 *   tnmc_sample call).  ckpt_stride = 0: keep the full environment stack (all L rows of every
 *   disorder).  ckpt_stride = k >= 1: keep only every k-th row plus one k-row
 *   segment and recompute segments inside tnmc_sample (the paper's "streaming protocol",
 *   PAPER.md:276, done by recomputation instead of disk).  Returns 0 on invalid arguments. */
size_t tnmc_workspace_bytes(int L, int chi, int n_dis, int n_samples_max, tnmc_prec prec,
                            int ckpt_stride);

/* Create a context for n_dis disorder realisations.
 *   Jr, Jd      [dev] int8 (n_dis, L, L), values in {-1, 0, +1}; read (bit-packed into the
 *               workspace) by a kernel enqueued on the stream; may be freed once the stream has
 *               passed that point.  Values outside {-1,0,+1} are treated as their sign (the values live on the device
 *               and are not read back: no TNMC_EINVAL for them); entries across the open boundary (Jr at c = L-1, Jd
 *               at r = L-1) are ignored.
 *   first_disorder  global index of disorder 0 (enters the Philox counter only)
 *   workspace   [dev] >= tnmc_workspace_bytes(...) bytes, 256-byte aligned
 *   cuda_stream a cudaStream_t (NULL = legacy default stream)
 * Errors: TNMC_EINVAL (L < 2, chi < 2 or > 32, non-finite or negative beta, null pointers,
 * misaligned workspace), TNMC_ENOMEM (workspace_bytes too small), TNMC_ECUDA. */
tnmc_status tnmc_create(tnmc_ctx** out, int L, int chi, double beta, int n_dis,
                        const int8_t* Jr, const int8_t* Jd, uint64_t first_disorder,
                        int n_samples_max, tnmc_prec prec, int ckpt_stride,
                        void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Real-valued couplings (Gaussian Edwards-Anderson and any other J_ij; SURVEY 8f NEXT-1 -- Eq. 1, Eq. 7 and
 * the whole method hold for any J_ij).  As tnmc_create, with
 *   Jr, Jd [dev] double (n_dis, L, L), 0 on the open boundary (c = L-1 for Jr, r = L-1 for Jd); copied into the
 *   workspace (>= tnmc_workspace_bytes_real) by a device-to-device copy enqueued on the stream.
 * A context created this way uses tnmc_energy_real / tnmc_metropolis_real (energies are doubles);
 * tnmc_energy returns TNMC_ESTATE on it (and tnmc_energy_real on a +-J context).  Everything else is the same. */
size_t tnmc_workspace_bytes_real(int L, int chi, int n_dis, int n_samples_max, tnmc_prec prec, int ckpt_stride);
tnmc_status tnmc_create_real(tnmc_ctx** out, int L, int chi, double beta, int n_dis,
                             const double* Jr, const double* Jd, uint64_t first_disorder,
                             int n_samples_max, tnmc_prec prec, int ckpt_stride,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);
/* E [dev] double (dis_count, n_samples): -sum_<ij> J_ij s_i s_j in FP64, deterministic summation order. */
tnmc_status tnmc_energy_real(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                             const uint32_t* cfg_bits, double* E);
/* As tnmc_metropolis with double energies (E and cur_E). */
tnmc_status tnmc_metropolis_real(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                                 const double* E, const double* logq,
                                 uint64_t seed, uint64_t step_offset,
                                 double* cur_logq, double* cur_E, int64_t* cur_idx,
                                 uint8_t* accepted, int64_t* n_accepted, double* sum_min1);

/* Build the boundary-MPS environment stack (steps a-1..a-7 of DESIGN.md).
 *   logZ [dev] double (n_dis) or NULL:  log Z_chi(d) = logscale_0 + log sum_sigma Psihat_0(sigma).
 * With ckpt_stride > 0 only the checkpoint rows are kept.  Must precede tnmc_sample. */
tnmc_status tnmc_build_envs(tnmc_ctx* ctx, double* logZ);

/* Draw n_samples configurations for each of disorders [dis_begin, dis_begin + dis_count).
 *   seed, sample_offset  Philox indexing (see above)
 *   cfg_bits [dev] uint32 (dis_count, n_samples, L, W)   out
 *   logq     [dev] double (dis_count, n_samples)         out: log q(s)
 * Errors: TNMC_ESTATE before tnmc_build_envs; TNMC_EINVAL on a bad range or
 * n_samples > n_samples_max. */
tnmc_status tnmc_sample(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                        uint64_t seed, uint64_t sample_offset,
                        uint32_t* cfg_bits, double* logq);

/* As tnmc_sample, with the test hooks of DESIGN.md:
 *   forced_cfg_bits [dev] uint32, same shape as cfg_bits, or NULL.  Teacher forcing: use these
 *                   spins instead of u < p; log q and probs are still those of the model
 *                   (cfg_bits receives a copy of the forced spins).
 *   probs           [dev] double (dis_count, n_samples, L, L) or NULL: q(s_i = +1 | s_<i). */
tnmc_status tnmc_sample_ex(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                           uint64_t seed, uint64_t sample_offset,
                           const uint32_t* forced_cfg_bits,
                           uint32_t* cfg_bits, double* logq, double* probs);

/* tnmc_sample with the energy (Eq. 1) and the magnetisation M = sum_i s_i of every drawn configuration
 * accumulated inside the left sampling sweep (the lane that packs a finished word of the new row also holds the word
 * above it: XOR + popcount against the coupling masks, the arithmetic of tnmc_energy), so that no second pass over
 * the configurations is needed -- and the configurations need not be stored at all:
 *   cfg_bits [dev] as tnmc_sample, or NULL: do not keep the configurations (at configs[4] they are 131 GB packed;
 *            E, M and log q are what the Metropolis scan and the thermal averages of E and M consume)
 *   E, M     [dev] int32 (dis_count, n_samples)  out; bit-identical to tnmc_energy / tnmc_observables' M on the same spins
 * +-J contexts only (TNMC_ESTATE on real couplings).  Other arguments and errors as tnmc_sample. */
tnmc_status tnmc_sample_fused(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                              uint64_t seed, uint64_t sample_offset,
                              uint32_t* cfg_bits, double* logq, int32_t* E, int32_t* M);

/* Exact energies, Eq. 1:  E = -sum_<ij> J_ij s_i s_j, integer arithmetic on the
 * packed words (XOR + popcount).
 *   cfg_bits [dev] uint32 (dis_count, n_samples, L, W)   in
 *   E        [dev] int32  (dis_count, n_samples)         out */
tnmc_status tnmc_energy(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                        const uint32_t* cfg_bits, int32_t* E);

/* Independence Metropolis scan, Eq. 10 (readings G15/G16): one chain per
 * disorder, proposals in sample order; accept iff log u < -beta (E' - E) + log q(s) - log q(s').
 *   E, logq     [dev] (dis_count, n_samples)  proposals
 *   seed, step_offset  Philox indexing: draw n of this call uses step index step_offset + n
 *   cur_logq, cur_E, cur_idx [dev] (dis_count)  in/out chain state; cur_idx < 0 means empty:
 *               the first proposal then initialises the chain (flag 1, not counted)
 *   accepted    [dev] uint8 (dis_count, n_samples)  out
 *   n_accepted  [dev] int64 (dis_count)  out: acceptances of this call
 *   sum_min1    [dev] double (dis_count) or NULL  out: sum over counted proposals of min(1, ratio) */
tnmc_status tnmc_metropolis(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                            const int32_t* E, const double* logq,
                            uint64_t seed, uint64_t step_offset,
                            double* cur_logq, int32_t* cur_E, int64_t* cur_idx,
                            uint8_t* accepted, int64_t* n_accepted, double* sum_min1);

/* Thermal averages along the Metropolis chain (the purpose of the samples; no code in the
 * paper; reading G19 of DESIGN.md): at step n the chain sits on the last accepted proposal and every step
 * counts once.  Per disorder the five sums over the steps of this call of  E, E^2, M, |M|, M^2  are ADDED
 * to `sums` (M = sum_i s_i; exact integer arithmetic, converted to double once per call).
 *   cfg_bits, E  [dev] as produced by tnmc_sample / tnmc_energy;  accepted [dev] uint8 from tnmc_metropolis
 *   M        [dev] int32 (dis_count, n_samples)  out: magnetisation of every proposal
 *   cur_E, cur_M [dev] int32 (dis_count)  in/out: state of the chain entering / leaving this call (read
 *            only while no proposal of the call has been accepted yet; a fresh chain's first flag is 1)
 *   sums     [dev] double (dis_count, 5)  in/out accumulators (zero them before the first call) */
tnmc_status tnmc_observables(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                             const uint32_t* cfg_bits, const int32_t* E, const uint8_t* accepted,
                             int32_t* M, int32_t* cur_E, int32_t* cur_M, double* sums);

/* As tnmc_observables for a context with real couplings: E and cur_E are doubles, the sums of E and E^2 are
 * FP64 sums in proposal order. */
tnmc_status tnmc_observables_real(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                                  const uint32_t* cfg_bits, const double* E, const uint8_t* accepted,
                                  int32_t* M, double* cur_E, int32_t* cur_M, double* sums);

/* Replica overlap along two independent Metropolis chains a, b of the same disorders (the spin-glass order
 * parameter: <M> = 0 by symmetry in the +-J model of PAPER.md:282-286, the overlap q = sum_i s_i^a s_i^b between two
 * replicas is the observable that carries the physics; no code in the paper; reading G19 of
 * DESIGN.md as for tnmc_observables): at step n each chain sits on its last accepted proposal and
 * q_n = N - 2 popcount(a xor b), an exact integer in [-N, N].
 *   cfg_a, accepted_a  [dev] proposals of chain a (dis_count, n_samples, L, W) and its flags from tnmc_metropolis
 *   cfg_b, accepted_b  [dev] likewise for chain b (e.g. a second tnmc_sample range of the same context)
 *   cur_cfg_a, cur_cfg_b [dev] uint32 (dis_count, L, W) in/out: state of each chain entering / leaving the call
 *               (read only for steps before that chain's first accepted proposal of this call; a fresh chain's first
 *               flag is 1, so fresh chains never read them)
 *   q_steps  [dev] int32 (dis_count, n_samples)  out: q_n of every step
 *   sums     [dev] double (dis_count, 3)  in/out: sum q, sum |q|, sum q^2 over the steps are ADDED (zero them first)
 * Both chains must cover the same disorders in the same order; works for +-J and real couplings alike. */
tnmc_status tnmc_replica_overlap(tnmc_ctx* ctx, int dis_count, int n_samples,
                                 const uint32_t* cfg_a, const uint8_t* accepted_a,
                                 const uint32_t* cfg_b, const uint8_t* accepted_b,
                                 uint32_t* cur_cfg_a, uint32_t* cur_cfg_b, int32_t* q_steps, double* sums);

/* tnmc_observables for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same two kernels, with the per-proposal magnetisations M -- the
 * scratch between them -- held in a file-scope device array of the library instead of a caller buffer.  The call
 * makes no cudaMalloc / cudaFree / allocating library call.  +-J contexts only.
 *   limit: dis_count * n_samples <= tnmc_observables_static_max() (2^20 proposals; the array is 4 MiB of device
 *   memory on every GPU that loads the library, held until exit).  Larger calls return TNMC_EINVAL.
 *   cfg_bits, E, accepted, cur_E, cur_M, sums: as tnmc_observables (no M output).
 * All calls on one device share the array: calls that may overlap on the GPU (different streams, no ordering) race.
 * Nothing in it has to start at zero -- each call overwrites the entries it reads. */
size_t tnmc_observables_static_max(void);
tnmc_status tnmc_observables_static(tnmc_ctx* ctx, int dis_begin, int dis_count, int n_samples,
                                    const uint32_t* cfg_bits, const int32_t* E, const uint8_t* accepted,
                                    int32_t* cur_E, int32_t* cur_M, double* sums);

/* One whole pass for host callers: copies Jr/Jd (host, int8 (n_dis,L,L)) to the device, builds
 * the environments, samples, computes energies, runs the Metropolis scan on fresh chains and
 * copies the results back.  All device memory comes from `workspace`
 * (>= tnmc_run_host_workspace_bytes).  Synchronises the stream before returning.
 *   out_cfg_bits [host] uint32 (n_dis, n_samples, L, W) or NULL
 *   out_E [host] int32, out_logq [host] double, out_accepted [host] uint8: (n_dis, n_samples)
 *   out_logZ [host] double (n_dis), out_n_accepted [host] int64 (n_dis); any may be NULL. */
size_t tnmc_run_host_workspace_bytes(int L, int chi, int n_dis, int n_samples, tnmc_prec prec,
                                     int ckpt_stride);
tnmc_status tnmc_run_host(int L, int chi, double beta, int n_dis, int n_samples,
                          const int8_t* Jr_host, const int8_t* Jd_host, uint64_t first_disorder,
                          uint64_t seed, tnmc_prec prec, int ckpt_stride,
                          void* workspace, size_t workspace_bytes, void* cuda_stream,
                          uint32_t* out_cfg_bits, int32_t* out_E, double* out_logq,
                          uint8_t* out_accepted, double* out_logZ, int64_t* out_n_accepted);

/* Device fault counters -> host_flags_out[TNMC_N_FLAGS] [host].  Synchronises the stream. */
tnmc_status tnmc_get_flags(tnmc_ctx* ctx, uint64_t* host_flags_out);

/* Test/inspection hook: copy one stored environment row of one disorder to the host in the
 * paper's layout: out [host] double (L, chi, 2, chi), zero-padded where the bond
 * is smaller than chi; *logscale_out [host] receives logscale_r (Psi_r = e^logscale Psihat_r).
 * TNMC_ESTATE if that row is not currently stored (checkpoint mode).  Synchronises. */
tnmc_status tnmc_get_env_row(tnmc_ctx* ctx, int disorder, int row, double* out,
                             double* logscale_out);

/* Roofline denominator probe: runs a register-resident FP64 microbenchmark on the current device
 * (148 x 2 CTAs of 256 threads, 8 independent chains per thread) for a few milliseconds and
 * returns the sustained rate in TFLOP/s: which = 0 -> scalar DFMA, which = 1 -> mma.sync.m8n8k4.f64
 * (DMMA).  scratch [dev] >= 1 MiB.  Synchronises.  Returns a negative value on a CUDA error. */
double tnmc_fp64_peak_tflops(int which, void* scratch, void* cuda_stream);

/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
uint64_t tnmc_launch_count(const tnmc_ctx* ctx);

const char* tnmc_last_error(const tnmc_ctx* ctx); /* never NULL; ctx may be NULL */
void tnmc_destroy(tnmc_ctx* ctx);                 /* frees host metadata only */

#ifdef __cplusplus
}
#endif
#endif /* TNMC_H_ */
