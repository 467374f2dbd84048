// pct_internal.h -- types shared by the kernels (pct_kernels.cu) and the C-ABI host code (pct_api.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "pct_rule.cuh"

namespace pct {

// Borrowed (or library-owned, for the host entry point) device arrays of the histories, include/pct.h.
struct HistPtrs {
    const float *t_in, *v_in, *t_out, *v_out, *dt_in, *dv_in, *dt_out, *dv_out, *wepl;
    const uint16_t* proj;
    const float *pcos, *psin;  // library-owned copies of the caller's tables
    int n_proj;
};

// Device-resident control block: lets every (accumulate, update) launch pair of a sweep use the
// SAME kernel arguments (so the pair can be replayed from a CUDA graph): the DROP block index
// lives here and is advanced by the update kernel.
struct Ctrl {
    unsigned long long work;      // next batch of the dynamic work queue of the accumulate kernel
    long long block;              // index of the DROP block the next accumulate launch processes
    unsigned long long cur[4];    // running counters of the current sweep: rows, nnz, segments, histories
    unsigned long long last[4];   // counters of the last completed sweep
};

struct DropArgs {
    Geom g;
    HistPtrs H;
    long long n;           // histories
    long long block_size;  // DROP block size
    long long first;       // >= 0: explicit range [first, first+count) (inspection); < 0: block from ctrl
    long long count;
    const float* x;        // image
    float2* acc;           // (Delta_j, c_j) interleaved
    const float4* tab;     // Sigma1^-1 table, nmin+1 entries
    Ctrl* ctrl;
    const uint32_t* order; // block mode: order[b*block_size + r] = offset inside DROP block b of the r-th
                           // history to process (k_order_blocks); nullptr: the caller's order
    float2* scratch;       // exact-traversal mode (pct_exact.cu): runs of every lane, cap_lane entries per lane; else nullptr
    int cap_lane;
};

struct RowsArgs {
    Geom g;
    HistPtrs H;
    long long first, count;
    int max_seg;
    const float4* tab;
    int32_t *nseg, *nnz, *seg_idx;
    float *seg_len, *row_len, *nodes;
};

// exact-traversal mode (pct_exact.cu)
size_t exact_scratch_bytes(int kmax, int grid, int* cap_lane_out);
cudaError_t exact_configure(int kmax);
cudaError_t launch_drop_exact(const DropArgs& a, int grid, cudaStream_t stream);
cudaError_t launch_rows_exact(const RowsArgs& a, int sms, cudaStream_t stream);

// launchers (pct_kernels.cu); all asynchronous on `stream`, return the launch error
size_t drop_smem_bytes(int nmin);
void bounds_dump(const char* tag);  // (a no-op unless built with -DPCT_CHECK_BOUNDS)
cudaError_t drop_configure(int nmin, int* grid_out);
cudaError_t launch_drop_block(const DropArgs& a, int grid, cudaStream_t stream);
cudaError_t launch_update(float* x, float2* acc, long long n_voxels, float lambda, Ctrl* ctrl,
                          long long n_blocks, bool top_down, cudaStream_t stream);
cudaError_t launch_split_acc(float2* acc, float* delta, float* cnt, const Geom& g, cudaStream_t stream);
cudaError_t launch_xyz_to_beam(float u_pl, long long n, const float* x, const float* y, const float* z, const float* tht, const float* thv,
                               const uint16_t* proj, const float* pcos, const float* psin, int n_proj, float* t_out, float* v_out,
                               cudaStream_t stream);
cudaError_t launch_image_io(float* x, float* ext, const Geom& g, bool to_storage, cudaStream_t stream);
cudaError_t launch_rows(const RowsArgs& a, bool pair_walk, cudaStream_t stream);
bool pair_enabled(int kmax);  // the two-histories-per-warp kernel serves this node count
cudaError_t launch_sum_stats(unsigned long long* dst, const unsigned long long* src, size_t pitch, int n_strings, cudaStream_t stream);
cudaError_t launch_rule_sweep(int which, uint32_t lo, uint32_t hi, unsigned long long* out, cudaStream_t stream);
cudaError_t launch_mean(float* x, const float* xs, int n_strings, long long n_voxels, long long pitch, cudaStream_t stream);
cudaError_t launch_order_blocks(const HistPtrs& H, const Geom& g, long long n, long long block_size, long long first_block,
                                long long n_blocks, int n_slabs, uint32_t* order, cudaStream_t stream);

// ---- total-variation superiorization (pct_tvs.cu) ---------------------------------------------------------------
constexpr int kTvMaxLevels = 8;
struct TvSums {
    double tvx, g2;              // TV(x) and ||grad TV(x)||^2
    double tvz[kTvMaxLevels];    // TV(x + beta 2^-l v)
};
struct TvState {
    TvSums sums[2];              // sums[parity] of the step in progress; the step zeroes the other pair for the next one
    double tv_before, tv_after;  // of the last completed step
    float beta[2];               // beta[parity]: step size of the step in progress; the other slot receives the next one
    float beta_used;             // step of the last completed step (beta 2^-level, or beta 2^-n_half if none was accepted)
    int level;                   // level accepted by the last step, -1: none
    unsigned int steps, accepted;
};
cudaError_t launch_tvs_step(float* x, float* grad, const Geom& g, long long n_slots, TvState* st, int parity, int n_half, float gamma,
                            int sms, cudaStream_t stream);

}  // namespace pct
