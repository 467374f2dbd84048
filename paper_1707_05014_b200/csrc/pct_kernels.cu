// pct_kernels.cu -- CUDA kernels of the pCT hot path for sm_100a.
//
//   k_drop_block  fused: history stream -> hull -> MLP -> voxel walk -> a_i.x, ||a_i||^2, residual
//                 -> scatter of (r_i a_ij, 1) into the block accumulator (R12).
//                 One WARP walks one history: lane l owns segments l, l+32, ... (the MLP node at
//                 depth k*h is closed-form in k, there is no recurrence along the path), the row
//                 (voxel, length) is parked in shared memory between the dot-product pass and the
//                 scatter pass, so the path is computed once per sweep.
//   k_update      x_j += lambda * Delta_j / max(1, c_j); accumulator zeroed; DROP block index advanced.
//   k_rows        inspection: same device functions, rows written out instead of consumed.
#include "pct_internal.h"

namespace pct {

constexpr int kWarpsPerCta = 8;
constexpr int kThreads = kWarpsPerCta * 32;
constexpr int kBatch = 8;  // histories a warp takes from the work queue per trip

__host__ __device__ inline int row_capacity(int nmin) { return (nmin + 2 + 3) & ~3; }
__host__ __device__ inline int tab_capacity(int nmin) { return (nmin + 1 + 3) & ~3; }

size_t drop_smem_bytes(int nmin) {
    const size_t per_warp = sizeof(PathState) * kBatch + 3 * sizeof(float) * row_capacity(nmin);
    return sizeof(float4) * tab_capacity(nmin) + kWarpsPerCta * per_warp;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ Hist load_history(const HistPtrs& H, long long i) {
    Hist hh;
    hh.t_in = __ldg(H.t_in + i);
    hh.v_in = __ldg(H.v_in + i);
    hh.t_out = __ldg(H.t_out + i);
    hh.v_out = __ldg(H.v_out + i);
    hh.dt_in = __ldg(H.dt_in + i);
    hh.dv_in = __ldg(H.dv_in + i);
    hh.dt_out = __ldg(H.dt_out + i);
    hh.dv_out = __ldg(H.dv_out + i);
    hh.wepl = __ldg(H.wepl + i);
    int p = (int)__ldg(H.proj + i);
    p = p < H.n_proj ? p : H.n_proj - 1;
    hh.cs = __ldg(H.pcos + p);
    hh.sn = __ldg(H.psin + p);
    return hh;
}

// Walk of one history by one warp (steps 3-4 of the rule): fills sidx/slen[0..K] in shared
// memory, returns this lane's part of the dot product a_i.x (x == nullptr: no gather).
// nodes_out (inspection only): (K+2) x 3 floats.
__device__ __forceinline__ float walk_history(const Geom& g, const PathState& S, const float4* __restrict__ tab,
                                              const float* __restrict__ x, int* sidx, float* slen, int lane,
                                              float* nodes_out) {
    const int K = S.K;
    float3 cur = node_position(g, S, tab, lane);
    float dot = 0.0f, pend_len = 0.0f, pend_x = 0.0f;
    for (int base = 0; base <= K; base += 32) {
        float3 nxt = cur;
        if (base + 32 <= K + 1) nxt = node_position(g, S, tab, base + 32 + lane);  // warp-uniform
        float3 up;
        up.x = __shfl_down_sync(0xffffffffu, cur.x, 1);
        up.y = __shfl_down_sync(0xffffffffu, cur.y, 1);
        up.z = __shfl_down_sync(0xffffffffu, cur.z, 1);
        const float n0x = __shfl_sync(0xffffffffu, nxt.x, 0);
        const float n0y = __shfl_sync(0xffffffffu, nxt.y, 0);
        const float n0z = __shfl_sync(0xffffffffu, nxt.z, 0);
        if (lane == 31) { up.x = n0x; up.y = n0y; up.z = n0z; }
        const int k = base + lane;
        int lin = -1;
        float len = 0.0f;
        if (k <= K) {
            segment(g, cur, up, lin, len);
            sidx[k] = lin;
            slen[k] = len;
        }
        if (nodes_out != nullptr && k <= K + 1) {
            nodes_out[3 * k + 0] = cur.x;
            nodes_out[3 * k + 1] = cur.y;
            nodes_out[3 * k + 2] = cur.z;
        }
        // the gather of the previous round is consumed only now: one round of independent work
        // sits between a load and its use
        dot = __fmaf_rn(pend_len, pend_x, dot);
        pend_len = len;
        pend_x = (x != nullptr && lin >= 0) ? x[lin] : 0.0f;
        cur = nxt;
    }
    if (nodes_out != nullptr && ((K + 1) & 31) == 0 && lane == 0) {  // node K+1 fell into a round of its own
        nodes_out[3 * (K + 1) + 0] = cur.x;
        nodes_out[3 * (K + 1) + 1] = cur.y;
        nodes_out[3 * (K + 1) + 2] = cur.z;
    }
    return __fmaf_rn(pend_len, pend_x, dot);
}

// Merge consecutive equal voxels (R10): slm[k] = merged chord length at the first segment of a
// run, 0 elsewhere (and for dropped segments).  Returns this lane's part of ||a_i||^2; nnz_lane
// counts this lane's run heads.
__device__ __forceinline__ float merge_runs(const int* sidx, const float* slen, float* slm, int K, int lane, int& nnz_lane) {
    float nrm = 0.0f;
    nnz_lane = 0;
    for (int k = lane; k <= K; k += 32) {
        const int idx = sidx[k];
        float lm = 0.0f;
        if (idx >= 0 && (k == 0 || sidx[k - 1] != idx)) {
            lm = slen[k];
            for (int m = k + 1; m <= K && sidx[m] == idx; ++m) lm += slen[m];
            nrm = __fmaf_rn(lm, lm, nrm);
            ++nnz_lane;
        }
        slm[k] = lm;
    }
    return nrm;
}

__global__ void __launch_bounds__(kThreads, 2) k_drop_block(const DropArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cap = row_capacity(g.nmin);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    unsigned char* wbase = smem_raw + sizeof(float4) * tab_capacity(g.nmin) +
                           (size_t)warp * (sizeof(PathState) * kBatch + 3 * sizeof(float) * cap);
    PathState* s_state = reinterpret_cast<PathState*>(wbase);
    int* sidx = reinterpret_cast<int*>(wbase + sizeof(PathState) * kBatch);
    float* slen = reinterpret_cast<float*>(sidx + cap);
    float* slm = slen + cap;

    for (int k = threadIdx.x; k <= g.nmin; k += kThreads) s_tab[k] = a.tab[k];
    __syncthreads();

    long long first = a.first, count = a.count;
    if (first < 0) {
        first = a.ctrl->block * a.block_size;
        count = a.n - first < a.block_size ? a.n - first : a.block_size;
    }
    const unsigned long long n_batches = (unsigned long long)((count + kBatch - 1) / kBatch);
    unsigned long long rows = 0, nnz = 0, segs = 0;

    for (;;) {
        unsigned long long b = 0;
        if (lane == 0) b = atomicAdd(&a.ctrl->work, 1ULL);
        b = __shfl_sync(0xffffffffu, b, 0);
        if (b >= n_batches) break;
        const long long i0 = first + (long long)b * kBatch;
        if (lane < kBatch) {
            const long long i = i0 + lane;
            if (i < first + count) {
                const Hist hh = load_history(a.H, i);
                setup_history(g, hh, s_state[lane]);
            } else {
                s_state[lane].K = -1;
            }
        }
        __syncwarp();
        for (int p = 0; p < kBatch; ++p) {
            const PathState& S = s_state[p];
            const int K = S.K;
            if (K < 0) continue;  // skipped history: empty row (R7)
            float dot = walk_history(g, S, s_tab, a.x, sidx, slen, lane, nullptr);
            __syncwarp();
            int nnz_lane;
            float nrm = merge_runs(sidx, slen, slm, K, lane, nnz_lane);
            dot = warp_sum(dot);
            nrm = warp_sum(nrm);
            if (nrm > 0.0f) {  // non-empty row (R13)
                const float r = __fdiv_rn(S.wepl - dot, nrm);
                for (int k = lane; k <= K; k += 32) {
                    const float lm = slm[k];
                    if (lm > 0.0f) atomicAdd(a.acc + sidx[k], make_float2(r * lm, 1.0f));
                }
                rows += (lane == 0);
                nnz += nnz_lane;
            }
            segs += (lane == 0) ? (K + 1) : 0;
            __syncwarp();  // the row buffers are reused by the next history
        }
        __syncwarp();  // the state records are reused by the next batch
    }
    nnz = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)nnz);
    if (lane == 0) {
        atomicAdd(&a.ctrl->cur[0], rows);
        atomicAdd(&a.ctrl->cur[1], nnz);
        atomicAdd(&a.ctrl->cur[2], segs);
    }
}

cudaError_t drop_configure(int nmin, int* grid_out) {
    const size_t smem = drop_smem_bytes(nmin);
    cudaError_t e = cudaFuncSetAttribute(k_drop_block, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_drop_block, kThreads, smem)) != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *grid_out = sms * per_sm;  // persistent: every CTA slot of the chip, work handed out dynamically
    return cudaSuccess;
}

cudaError_t launch_drop_block(const DropArgs& a, int grid, cudaStream_t stream) {
    // never more CTAs than batches of work (small blocks: fewer, fuller CTAs start faster)
    const long long cnt = a.first < 0 ? a.block_size : a.count;
    const long long need = (cnt + (long long)kBatch * kWarpsPerCta - 1) / ((long long)kBatch * kWarpsPerCta);
    if (need < grid) grid = need < 1 ? 1 : (int)need;
    k_drop_block<<<grid, kThreads, drop_smem_bytes(a.g.nmin), stream>>>(a);
    return cudaGetLastError();
}

// x_j += lambda * Delta_j / max(1, c_j) (R12); c_j >= 1 wherever anything was accumulated.
__device__ __forceinline__ float updated(float xv, float2 dc, float lambda) {
    return dc.y > 0.0f ? xv + __fdiv_rn(lambda * dc.x, dc.y) : xv;
}

__global__ void __launch_bounds__(256) k_update(float* __restrict__ x, float2* __restrict__ acc, long long n_voxels,
                                                float lambda, Ctrl* ctrl, long long n_blocks) {
    const long long n4 = n_voxels >> 2;
    const long long stride = (long long)gridDim.x * blockDim.x;
    float4* x4 = reinterpret_cast<float4*>(x);
    float4* a4 = reinterpret_cast<float4*>(acc);
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += stride) {
        const float4 a01 = a4[2 * q], a23 = a4[2 * q + 1];
        const bool hit01 = a01.y > 0.0f || a01.w > 0.0f, hit23 = a23.y > 0.0f || a23.w > 0.0f;
        if (hit01 || hit23) {
            float4 xv = x4[q];
            xv.x = updated(xv.x, make_float2(a01.x, a01.y), lambda);
            xv.y = updated(xv.y, make_float2(a01.z, a01.w), lambda);
            xv.z = updated(xv.z, make_float2(a23.x, a23.y), lambda);
            xv.w = updated(xv.w, make_float2(a23.z, a23.w), lambda);
            x4[q] = xv;
            const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
            if (hit01) a4[2 * q] = z;
            if (hit23) a4[2 * q + 1] = z;
        }
    }
    if (blockIdx.x == 0) {
        for (long long j = (n4 << 2) + threadIdx.x; j < n_voxels; j += blockDim.x) {  // ragged tail
            const float2 dc = acc[j];
            if (dc.y > 0.0f) {
                x[j] = updated(x[j], dc, lambda);
                acc[j] = make_float2(0.f, 0.f);
            }
        }
        if (threadIdx.x == 0 && ctrl != nullptr) {
            ctrl->work = 0ULL;
            const long long nb = ctrl->block + 1;
            if (nb >= n_blocks) {  // sweep complete: publish its counters
                for (int s = 0; s < 4; ++s) {
                    ctrl->last[s] = ctrl->cur[s];
                    ctrl->cur[s] = 0ULL;
                }
                ctrl->block = 0;
            } else {
                ctrl->block = nb;
            }
        }
    }
}

cudaError_t launch_update(float* x, float2* acc, long long n_voxels, float lambda, Ctrl* ctrl, long long n_blocks,
                          cudaStream_t stream) {
    const long long n4 = n_voxels >> 2;
    long long blocks = (n4 + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_update<<<(int)blocks, 256, 0, stream>>>(x, acc, n_voxels, lambda, ctrl, n_blocks);
    return cudaGetLastError();
}

// inspection: de-interleave the accumulator into Delta and c, and zero it
__global__ void k_split_acc(float2* __restrict__ acc, float* __restrict__ delta, float* __restrict__ cnt, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        const float2 dc = acc[j];
        delta[j] = dc.x;
        cnt[j] = dc.y;
        acc[j] = make_float2(0.f, 0.f);
    }
}

cudaError_t launch_split_acc(float2* acc, float* delta, float* cnt, long long n, cudaStream_t stream) {
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_split_acc<<<(int)blocks, 256, 0, stream>>>(acc, delta, cnt, n);
    return cudaGetLastError();
}

// inspection: one warp per history, rows written out (include/pct.h, pct_debug_rows)
__global__ void __launch_bounds__(kThreads) k_rows(const RowsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cap = row_capacity(g.nmin);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    unsigned char* wbase = smem_raw + sizeof(float4) * tab_capacity(g.nmin) +
                           (size_t)warp * (sizeof(PathState) * kBatch + 3 * sizeof(float) * cap);
    PathState* s_state = reinterpret_cast<PathState*>(wbase);
    int* sidx = reinterpret_cast<int*>(wbase + sizeof(PathState) * kBatch);
    float* slen = reinterpret_cast<float*>(sidx + cap);
    float* slm = slen + cap;
    for (int k = threadIdx.x; k <= g.nmin; k += kThreads) s_tab[k] = a.tab[k];
    __syncthreads();
    for (long long r = (long long)blockIdx.x * kWarpsPerCta + warp; r < a.count; r += (long long)gridDim.x * kWarpsPerCta) {
        if (lane == 0) {
            const Hist hh = load_history(a.H, a.first + r);
            setup_history(g, hh, s_state[0]);
        }
        __syncwarp();
        const PathState& S = s_state[0];
        const int K = S.K;
        int nnz_total = 0;
        if (K >= 0) {
            float* nodes = a.nodes ? a.nodes + (size_t)r * (a.max_seg + 1) * 3 : nullptr;
            walk_history(g, S, s_tab, nullptr, sidx, slen, lane, nodes);
            __syncwarp();
            int nnz_lane;
            merge_runs(sidx, slen, slm, K, lane, nnz_lane);
            nnz_total = __reduce_add_sync(0xffffffffu, nnz_lane);
            for (int k = lane; k <= K; k += 32) {
                const size_t o = (size_t)r * a.max_seg + k;
                if (a.seg_idx) a.seg_idx[o] = sidx[k];
                if (a.seg_len) a.seg_len[o] = slen[k];
                if (a.row_len) a.row_len[o] = slm[k];
            }
        }
        if (lane == 0) {
            a.nseg[r] = K >= 0 ? K + 1 : 0;
            a.nnz[r] = nnz_total;
        }
        __syncwarp();
    }
}

cudaError_t launch_rows(const RowsArgs& a, cudaStream_t stream) {
    const size_t smem = drop_smem_bytes(a.g.nmin);
    cudaError_t e = cudaFuncSetAttribute(k_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    long long blocks = (a.count + kWarpsPerCta - 1) / kWarpsPerCta;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    k_rows<<<(int)blocks, kThreads, smem, stream>>>(a);
    return cudaGetLastError();
}

}  // namespace pct
