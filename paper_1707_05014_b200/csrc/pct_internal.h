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

// launchers (pct_kernels.cu); all asynchronous on `stream`, return the launch error
size_t drop_smem_bytes(int nmin);
cudaError_t drop_configure(int nmin, int* grid_out);
cudaError_t launch_drop_block(const DropArgs& a, int grid, cudaStream_t stream);
cudaError_t launch_update(float* x, float2* acc, long long n_voxels, float lambda, Ctrl* ctrl,
                          long long n_blocks, cudaStream_t stream);
cudaError_t launch_split_acc(float2* acc, float* delta, float* cnt, long long n_voxels, cudaStream_t stream);
cudaError_t launch_rows(const RowsArgs& a, cudaStream_t stream);
cudaError_t launch_mean(float* x, const float* xs, int n_strings, long long n_voxels, cudaStream_t stream);
cudaError_t launch_order_blocks(const HistPtrs& H, const Geom& g, long long n, long long block_size, long long first_block,
                                long long n_blocks, int n_slabs, uint32_t* order, cudaStream_t stream);

}  // namespace pct
