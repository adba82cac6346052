// tnmc_ctx.cuh -- host-side context: workspace carve-up and the environment-stack policy (a-6).
#pragma once
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/tnmc.h"
#include "tnmc_build.cuh"
#include "tnmc_common.cuh"
#include "tnmc_energy.cuh"
#include "tnmc_sample.cuh"
#include "tnmc_sample_tf32.cuh"

namespace tnmc {

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Environment-stack policy.
//   ckpt == 0: every row r lives in slot r.
//   ckpt == k: permanent slots hold rows 0, k, 2k, ... ("checkpoints") and the bottom row L-1;
//              max(k-1, 2) further slots hold the rows of the segment being sampled (and serve as
//              the ping-pong pair of the first pass).  Segment j = rows [jk, min((j+1)k, L)).
struct Plan {
    int L = 0, chi = 0, P = 0, W = 0, n_dis = 0, n_samples_max = 0, ckpt = 0;
    int f32 = 0;                    // environment stack stored in FP32 (TNMC_F32_LOGSCALE, TNMC_F32_STORE)
    int tf32 = 0;                   // TF32 tensor-core sampler and its fragment order (TNMC_F32_LOGSCALE, TNMC_TF32_FAST)
    int x3 = 0;                     // error-compensated 3xTF32 products (TNMC_F32_LOGSCALE)
    int real_j = 0;                 // real-valued couplings kept as doubles (tnmc_create_real)
    int n_seg = 1, n_slots = 0, n_seg_slots = 0, n_maps = 1, tiles = 1;
    size_t tsz = 0;                 // doubles per site tensor
    size_t env_dis_stride = 0;      // doubles per disorder
    size_t qsz = 0;                 // doubles per site of the Q scratch
    // byte offsets into the workspace
    size_t off_masks = 0, off_maps = 0, off_flags = 0, off_logscale = 0, off_logz = 0, off_env = 0,
           off_qbuf = 0, off_m0 = 0, off_renv = 0, off_jreal = 0, off_carry = 0, total = 0;

    int ckpt_slot(int j) const { return j; }
    int bottom_slot() const { return n_seg; }
    int seg_slot(int i) const { return n_seg + 1 + i; }
    // permanent slot of row r, or -1
    int perm_slot(int r) const {
        if (ckpt == 0) return r;
        if (r == L - 1) return bottom_slot();
        if (r % ckpt == 0) return ckpt_slot(r / ckpt);
        return -1;
    }
    // slot map m (m == 0 first pass; m == 1 + j: segment j, checkpoint mode only): slot_maps_kernel below
    // first stored row at or below the end of segment j: where its recomputation starts
    int seg_start_row(int j) const { const int h = (j + 1) * ckpt; return h <= L - 1 ? h : L - 1; }
    int seg_end(int j) const { const int h = (j + 1) * ckpt; return h < L ? h : L; }
};

inline bool make_plan(Plan& p, int L, int chi, int n_dis, int n_samples_max, int ckpt, int prec = 0, int real_j = 0) {
    p.real_j = real_j;
    if (prec < 0 || prec > 3) return false;
    p.f32 = prec != 0;
    p.tf32 = prec == 1 || prec == 3;
    p.x3 = prec == 1;
    if (L < 2 || L > 4096 || chi < 2 || chi > 32 || n_dis < 1 || n_samples_max < 1 || ckpt < 0) return false;
    if (ckpt >= L) ckpt = 0;
    p.L = L; p.chi = chi; p.P = pad_chi(chi); p.W = (L + 31) / 32; p.n_dis = n_dis;
    p.n_samples_max = n_samples_max; p.ckpt = ckpt;
    p.tsz = (size_t)2 * p.P * p.P;
    if (ckpt == 0) { p.n_seg = 1; p.n_seg_slots = 0; p.n_slots = L; p.n_maps = 1; }
    else {
        p.n_seg = (L + ckpt - 1) / ckpt;
        p.n_seg_slots = ckpt - 1 > 2 ? ckpt - 1 : 2;
        p.n_slots = p.n_seg + 1 + p.n_seg_slots;
        p.n_maps = 1 + p.n_seg;
    }
    p.env_dis_stride = (size_t)p.n_slots * L * p.tsz;
    p.qsz = (size_t)(2 * p.P + 4) * (2 * p.P) + 4 * p.P;   // BuildCfg<P>::QSZ
    p.tiles = (n_samples_max + SAMPLE_CHAINS - 1) / SAMPLE_CHAINS;
    size_t o = 0;
    p.off_masks = o;    o = align_up(o + sizeof(uint32_t) * 4 * (size_t)n_dis * L * p.W);
    p.off_maps = o;     o = align_up(o + sizeof(int) * (size_t)p.n_maps * L);
    p.off_flags = o;    o = align_up(o + sizeof(unsigned long long) * N_FLAGS);
    p.off_logscale = o; o = align_up(o + sizeof(double) * (size_t)n_dis * L);
    p.off_logz = o;     o = align_up(o + sizeof(double) * (size_t)n_dis);
    p.off_env = o;      o = align_up(o + (p.f32 ? sizeof(float) : sizeof(double)) * (size_t)n_dis * p.env_dis_stride);
    p.off_qbuf = o;     o = align_up(o + sizeof(double) * (size_t)n_dis * L * p.qsz);
    p.off_m0 = o;       o = align_up(o + sizeof(double) * (size_t)n_dis * 4 * p.P * p.P);
    p.off_renv = o;     o = align_up(o + sizeof(double) * (size_t)n_dis * p.tiles * L * SAMPLE_CHAINS * p.P);
    p.off_jreal = o;    o = align_up(o + (real_j ? sizeof(double) * 2 * (size_t)n_dis * L * L : 0));
    // last row of a row range for tnmc_sample_fused without stored configurations (checkpoint mode only)
    p.off_carry = o;    o = align_up(o + (ckpt ? sizeof(uint32_t) * (size_t)n_dis * n_samples_max * p.W : 0));
    p.total = o;
    return true;
}

// The slot maps of a Plan, written on the device: maps[m][r] = slot of row r in pass m, -1 if row r is not held.
//   permanent slots (perm_slot above) first; pass 0 ping-pongs the other rows through the first two segment slots;
//   pass 1 + j holds the inner rows of segment j in the segment slots.
__global__ void slot_maps_kernel(int L, int ckpt, int n_seg, int n_maps, int* maps) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_maps * L) return;
    const int m = idx / L, r = idx - m * L;
    int s;
    if (ckpt == 0) s = r;
    else if (r == L - 1) s = n_seg;                       // bottom_slot
    else if (r % ckpt == 0) s = r / ckpt;                 // ckpt_slot
    else if (m == 0) s = n_seg + 1 + (r & 1);             // seg_slot(r & 1)
    else {
        const int j = m - 1;
        s = (r > j * ckpt && r < (j + 1) * ckpt) ? n_seg + 1 + (r - j * ckpt - 1) : -1;
    }
    maps[idx] = s;
}

}  // namespace tnmc

struct tnmc_ctx {
    tnmc::Plan plan;
    double beta = 0.0;
    uint64_t first_disorder = 0;
    cudaStream_t stream = nullptr;
    char* ws = nullptr;
    bool built = false;
    uint64_t launches = 0;
    std::string err;

    template <class T> T* at(size_t off) const { return reinterpret_cast<T*>(ws + off); }
    tnmc::JView jview() const {
        tnmc::JView v;
        v.masks = at<uint32_t>(plan.off_masks);
        v.jr_real = plan.real_j ? at<double>(plan.off_jreal) : nullptr;
        v.jd_real = plan.real_j ? at<double>(plan.off_jreal) + (size_t)plan.n_dis * plan.L * plan.L : nullptr;
        v.n_dis = plan.n_dis; v.L = plan.L; v.W = plan.W;
        return v;
    }
    const int* map(int m) const { return at<int>(plan.off_maps) + (size_t)m * plan.L; }
    tnmc::EnvRef env() const { tnmc::EnvRef e; e.base = ws + plan.off_env; e.f32 = plan.f32; e.lay32 = plan.tf32; return e; }
};
