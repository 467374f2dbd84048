// pct_kernels.cu -- CUDA kernels of the pCT hot path for sm_100a.
//
//   k_drop_block  fused: history stream -> hull -> MLP -> voxel walk -> a_i.x, ||a_i||^2, residual
//                 -> scatter of (r_i a_ij, 1) into the block accumulator (R12).
//                 One WARP walks one history; lane l owns the CONTIGUOUS chunk of segments
//                 [l*C, (l+1)*C), C = ceil((K+1)/32) (the MLP node at depth k*h is closed-form in
//                 k, there is no recurrence along the path).  A lane keeps its <= CMAX (voxel,
//                 length, x) triples in registers between the dot-product pass and the scatter
//                 pass, so the path is computed once per sweep and never touches memory; runs of
//                 equal voxels are merged sequentially inside a lane, and the at most 31 lane
//                 seams are patched with three shuffles.
//   k_update      x_j += lambda * Delta_j / max(1, c_j); accumulator zeroed; DROP block index advanced.
//   k_rows        inspection: the same walk, rows written out instead of consumed.
#include "pct_internal.h"

namespace pct {

constexpr int kWarpsPerCta = 8;
constexpr int kThreads = kWarpsPerCta * 32;
constexpr int kBatch = 8;  // histories a warp takes from the work queue per trip (at most)

// Sigma1^-1 table in shared memory: entry k sits at slot k + (k >> 3), so that the 8 lanes of a
// quarter warp, which read entries C apart, fall into different 16-byte bank groups for every
// chunk size C <= 9 (plain layout: C = 8 would be an 8-way conflict).  The table is padded with
// zero entries up to k = nmin + 32: lanes past the end of a path read (and discard) them.
__host__ __device__ inline int tab_slot(int k) { return k + (k >> 3); }
__host__ __device__ inline int tab_slots(int nmin) { return (tab_slot(nmin + 33) + 4) & ~3; }

size_t drop_smem_bytes(int nmin) {
    return sizeof(float4) * tab_slots(nmin) + (size_t)kWarpsPerCta * kBatch * sizeof(PathState);
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

__device__ __forceinline__ void stage_table(float4* s_tab, const float4* __restrict__ tab, int nmin) {
    const int n = tab_slots(nmin);
    for (int q = threadIdx.x; q < n; q += kThreads) s_tab[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    for (int k = threadIdx.x; k <= nmin; k += kThreads) s_tab[tab_slot(k)] = tab[k];
    __syncthreads();
}

// Where the inspection kernel wants the row of one history written (all optional).
struct EmitPtrs {
    int32_t* seg_idx;
    float *seg_len, *row_len, *nodes;
};

// One lane's part of the row of one history, in registers.
template <int CMAX>
struct LaneRow {
    int lin[CMAX];    // voxel of segment k0 + c, -1: outside the grid or past the end of the path
    float len[CMAX];  // its length, 0 where lin < 0
    unsigned heads;   // bit c: segment k0 + c starts a run of equal voxels (R10) = one non-zero of the row
    int C;            // segments per lane of this history
};

__device__ __forceinline__ void emit_segment(const EmitPtrs& em, int k, int K, int lin, float len, const float3 a,
                                             const float3 exitP) {
    if (em.seg_idx) em.seg_idx[k] = lin;
    if (em.seg_len) em.seg_len[k] = len;
    if (em.nodes) {
        em.nodes[3 * k + 0] = a.x;
        em.nodes[3 * k + 1] = a.y;
        em.nodes[3 * k + 2] = a.z;
        if (k == K) {
            em.nodes[3 * k + 3] = exitP.x;
            em.nodes[3 * k + 4] = exitP.y;
            em.nodes[3 * k + 5] = exitP.z;
        }
    }
}

// Walk of one history by one warp (steps 3-4 of the rule).  Fills the lane's part of the row,
// returns the lane's parts of a_i.x (GATHER), ||a_i||^2 and the non-zero count.
//
// Lane l evaluates the MLP at nodes k0+1 .. k0+C (k0 = l*C); its segment c joins nodes k0+c and
// k0+c+1, so segments 1..C-1 need only the lane's own nodes and segment 0 starts at the LAST node
// of lane l-1, fetched with one shuffle after the node loop (lane 0: the hull entry point).
// Lanes past the end of the path run the same instructions on harmless values and are masked.
template <int CMAX, bool GATHER, bool EMIT>
__device__ __forceinline__ void walk_history(const Geom& g, const PathState& S, const float4* s_tab,
                                             const float* __restrict__ x, int lane, LaneRow<CMAX>& row, float& dot,
                                             float& nrm, int& nnz, const EmitPtrs& em) {
    const PathState st = S;  // shared memory -> registers, once per history
    const int K = st.K;
    const int C = (K + 32) >> 5;  // ceil((K + 1) / 32) segments per lane
    const int k0 = lane * C;
    row.C = C;
    const float3 exitP = to_object(st, st.t2, st.u2, st.v2);  // node K+1: the hull exit point, assigned (R9)
    float xv[CMAX];
    float3 n1 = exitP, prv = exitP;
#pragma unroll
    for (int j = 1; j <= CMAX; ++j) {
        if (j < CMAX) {
            row.lin[j] = -1;
            row.len[j] = 0.0f;
            xv[j] = 0.0f;
        }
        if (j <= C) {  // warp-uniform
            const int k = k0 + j;  // node index
            float3 nd = mlp_node(g, st, s_tab[tab_slot(k)], k);
            if (k > K) nd = exitP;
            if (j == 1) {
                n1 = nd;
            } else {  // segment k-1 = slot j-1, between the lane's nodes j-1 and j
                int lin;
                float len;
                segment(g, prv, nd, lin, len);
                const bool ok = (k - 1 <= K) && lin >= 0;
                row.lin[j - 1] = ok ? lin : -1;
                row.len[j - 1] = ok ? len : 0.0f;
                if (GATHER) {
                    if (ok) xv[j - 1] = __ldg(x + lin);
                }
                if (EMIT) {
                    if (k - 1 <= K) emit_segment(em, k - 1, K, lin, len, prv, exitP);
                }
            }
            prv = nd;
        }
    }
    {  // slot 0: from the last node of the previous lane (= node k0) to the lane's first node
        float3 start;
        start.x = __shfl_up_sync(0xffffffffu, prv.x, 1);
        start.y = __shfl_up_sync(0xffffffffu, prv.y, 1);
        start.z = __shfl_up_sync(0xffffffffu, prv.z, 1);
        if (lane == 0) start = to_object(st, st.t0, st.u0, st.v0);  // node 0: the hull entry point (R9)
        int lin;
        float len;
        segment(g, start, n1, lin, len);
        const bool ok = (k0 <= K) && lin >= 0;
        row.lin[0] = ok ? lin : -1;
        row.len[0] = ok ? len : 0.0f;
        xv[0] = 0.0f;
        if (GATHER) {
            if (ok) xv[0] = __ldg(x + lin);
        }
        if (EMIT) {
            if (k0 <= K) emit_segment(em, k0, K, lin, len, start, exitP);
        }
    }
    // ---- a_i.x, and the merge of consecutive equal voxels (R10), sequential inside the lane ----
    dot = 0.0f;
    nrm = 0.0f;
    nnz = 0;
    unsigned heads = 0u;
    int run_idx = -2;        // voxel of the current run (-2: none yet)
    float run_len = 0.0f;    // its length so far (this lane's part)
    float first_len = 0.0f;  // length of the lane's first run (this lane's part)
    bool whole = true;       // the lane's whole chunk is one run
#pragma unroll
    for (int c = 0; c < CMAX; ++c) {
        if (c < C) {
            dot = __fmaf_rn(row.len[c], xv[c], dot);
            const bool fresh = row.lin[c] != run_idx;
            if (fresh) {
                nrm = __fmaf_rn(run_len, run_len, nrm);  // the finished run
                if (c > 0 && whole) {
                    first_len = run_len;
                    whole = false;
                }
                run_idx = row.lin[c];
                run_len = row.len[c];
                if (run_idx >= 0) {
                    heads |= 1u << c;
                    ++nnz;
                }
            } else {
                run_len += row.len[c];
            }
        }
    }
    nrm = __fmaf_rn(run_len, run_len, nrm);
    if (whole) first_len = run_len;
    // ---- lane seams: the lane's first run may continue the previous lane's last run ----------
    // With p = this lane's part and q = the part in earlier lanes, (q + p)^2 = q^2 + 2qp + p^2:
    // q^2 is already in the earlier lanes' sums, p^2 in this lane's, the seam adds 2qp.
    const int prev_idx = __shfl_up_sync(0xffffffffu, run_idx, 1);
    const float prev_len = __shfl_up_sync(0xffffffffu, run_len, 1);
    const bool prev_whole = __shfl_up_sync(0xffffffffu, (int)whole, 1) != 0;
    const bool cont = lane > 0 && row.lin[0] >= 0 && row.lin[0] == prev_idx;
    const float base = cont ? prev_len : 0.0f;
    float carry = base;  // length of the lane's first run that lies in earlier lanes
    if (__any_sync(0xffffffffu, cont && prev_whole)) {
        // a run spans three or more lanes (only when C <= 3): chase it through the whole-lane runs
        for (int it = 0; it < 31; ++it) {
            const float up = __shfl_up_sync(0xffffffffu, carry, 1);
            const float nc = (cont && prev_whole) ? base + up : base;
            const bool changed = nc != carry;
            carry = nc;
            if (!__any_sync(0xffffffffu, changed)) break;
        }
    }
    if (cont) {
        heads &= ~1u;
        --nnz;
        nrm = __fmaf_rn(2.0f * carry, first_len, nrm);
    }
    row.heads = heads;
    if (EMIT) {
        if (em.row_len) {
#pragma unroll
            for (int c = 0; c < CMAX; ++c)
                if (c < C && k0 + c <= K) em.row_len[k0 + c] = ((heads >> c) & 1u) ? 1.0f : 0.0f;
        }
    }
}

// Work queue of one DROP block: items of kBatch histories first, then (the last ~1/8 of the
// block) items of kBatch/4, so that the warps run dry within a couple of histories of each
// other.  Small blocks get smaller items so that they still spread over the whole grid.
struct Queue {
    long long first, count;
    int big, small;            // histories per item in the two phases
    unsigned long long n_big;  // items of the first phase
    unsigned long long n_items;
};

__device__ __forceinline__ Queue make_queue(long long first, long long count, long long n_warps) {
    Queue q;
    q.first = first;
    q.count = count;
    long long big = count / (4 * n_warps);
    big = big < 1 ? 1 : (big > kBatch ? kBatch : big);
    const long long small = big >= 4 ? big / 4 : 1;
    const long long nb = (count - count / 8) / big;
    const long long rest = count - nb * big;
    q.big = (int)big;
    q.small = (int)small;
    q.n_big = (unsigned long long)nb;
    q.n_items = (unsigned long long)(nb + (rest + small - 1) / small);
    return q;
}

template <int CMAX>
__global__ void __launch_bounds__(kThreads, 2) k_drop_block(const DropArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + sizeof(float4) * tab_slots(g.nmin)) + warp * kBatch;
    stage_table(s_tab, a.tab, g.nmin);

    long long first = a.first, count = a.count;
    if (first < 0) {
        first = a.ctrl->block * a.block_size;
        count = a.n - first < a.block_size ? a.n - first : a.block_size;
    }
    const Queue q = make_queue(first, count, (long long)gridDim.x * kWarpsPerCta);
    unsigned long long rows = 0, nnz_total = 0, segs = 0;
    const EmitPtrs no_emit{nullptr, nullptr, nullptr, nullptr};

    for (;;) {
        unsigned long long w = 0;
        if (lane == 0) w = atomicAdd(&a.ctrl->work, 1ULL);
        w = __shfl_sync(0xffffffffu, w, 0);
        if (w >= q.n_items) break;
        long long i0;
        int cnt;
        if (w < q.n_big) {
            i0 = q.first + (long long)w * q.big;
            cnt = q.big;
        } else {
            i0 = q.first + (long long)q.n_big * q.big + (long long)(w - q.n_big) * q.small;
            cnt = q.small;
        }
        const long long left = q.first + q.count - i0;
        if (left < cnt) cnt = (int)left;
        if (lane < cnt) {
            const Hist hh = load_history(a.H, i0 + lane);
            setup_history(g, hh, s_state[lane]);
        }
        __syncwarp();
        for (int p = 0; p < cnt; ++p) {
            const PathState& S = s_state[p];
            const int K = S.K;
            if (K < 0) continue;  // skipped history: empty row (R7)
            LaneRow<CMAX> row;
            float dot, nrm;
            int nnz;
            walk_history<CMAX, true, false>(g, S, s_tab, a.x, lane, row, dot, nrm, nnz, no_emit);
            dot = warp_sum(dot);
            nrm = warp_sum(nrm);
            if (nrm > 0.0f) {  // non-empty row (R13)
                const float r = __fdiv_rn(S.wepl - dot, nrm);
#pragma unroll
                for (int c = 0; c < CMAX; ++c) {
                    if (c < row.C && row.lin[c] >= 0)
                        atomicAdd(a.acc + row.lin[c], make_float2(r * row.len[c], ((row.heads >> c) & 1u) ? 1.0f : 0.0f));
                }
                rows += (lane == 0);
                nnz_total += nnz;
            }
            segs += (lane == 0) ? (K + 1) : 0;
        }
        __syncwarp();  // the state records are reused by the next item
    }
    nnz_total = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)nnz_total);
    if (lane == 0) {
        atomicAdd(&a.ctrl->cur[0], rows);
        atomicAdd(&a.ctrl->cur[1], nnz_total);
        atomicAdd(&a.ctrl->cur[2], segs);
    }
}

// Chunk capacities the kernels are instantiated for: CMAX >= ceil((nmin + 1) / 32).
#define PCT_FOR_CMAX(nmin, CALL)                  \
    do {                                          \
        const int cneed__ = ((nmin) + 32) >> 5;   \
        if (cneed__ <= 3) { CALL(3); }            \
        else if (cneed__ <= 5) { CALL(5); }       \
        else if (cneed__ <= 7) { CALL(7); }       \
        else if (cneed__ <= 9) { CALL(9); }       \
        else if (cneed__ <= 16) { CALL(16); }     \
        else { CALL(32); }                        \
    } while (0)

cudaError_t drop_configure(int nmin, int* grid_out) {
    if (((nmin + 32) >> 5) > 32) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(nmin);
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
#define PCT_CFG(CM)                                                                                                  \
    e = cudaFuncSetAttribute(k_drop_block<CM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);               \
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_drop_block<CM>, kThreads, smem)
    PCT_FOR_CMAX(nmin, PCT_CFG);
#undef PCT_CFG
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *grid_out = sms * per_sm;  // persistent: every CTA slot of the chip, work handed out dynamically
    return cudaSuccess;
}

cudaError_t launch_drop_block(const DropArgs& a, int grid, cudaStream_t stream) {
    // never more warps than histories (small blocks: one history per warp)
    const long long cnt = a.first < 0 ? a.block_size : a.count;
    const long long need = (cnt + kWarpsPerCta - 1) / kWarpsPerCta;
    if (need < grid) grid = need < 1 ? 1 : (int)need;
    const size_t smem = drop_smem_bytes(a.g.nmin);
#define PCT_LAUNCH(CM) k_drop_block<CM><<<grid, kThreads, smem, stream>>>(a)
    PCT_FOR_CMAX(a.g.nmin, PCT_LAUNCH);
#undef PCT_LAUNCH
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

// inspection: one warp per history, rows written out (include/pct.h, pct_debug_rows).  The walk,
// the run heads and the non-zero count are those of the hot path; only the merged length of a
// run (which the hot path never forms: it needs ||a_i||^2 and the unmerged scatter only) is
// summed here, from the segment lengths just written.
template <int CMAX>
__global__ void __launch_bounds__(kThreads) k_rows(const RowsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + sizeof(float4) * tab_slots(g.nmin)) + warp * kBatch;
    stage_table(s_tab, a.tab, g.nmin);
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
            EmitPtrs em;
            em.seg_idx = a.seg_idx ? a.seg_idx + (size_t)r * a.max_seg : nullptr;
            em.seg_len = a.seg_len ? a.seg_len + (size_t)r * a.max_seg : nullptr;
            em.row_len = a.row_len ? a.row_len + (size_t)r * a.max_seg : nullptr;
            em.nodes = a.nodes ? a.nodes + (size_t)r * (a.max_seg + 1) * 3 : nullptr;
            LaneRow<CMAX> row;
            float dot, nrm;
            int nnz;
            walk_history<CMAX, false, true>(g, S, s_tab, nullptr, lane, row, dot, nrm, nnz, em);
            nnz_total = __reduce_add_sync(0xffffffffu, nnz);
            __syncwarp();
            if (em.row_len && em.seg_idx && em.seg_len) {
                for (int k = lane; k <= K; k += 32) {
                    if (em.row_len[k] > 0.0f) {  // run head: add up the run
                        const int idx = em.seg_idx[k];
                        float lm = em.seg_len[k];
                        for (int m = k + 1; m <= K && em.seg_idx[m] == idx; ++m) lm += em.seg_len[m];
                        em.row_len[k] = lm;
                    }
                }
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
    if (((a.g.nmin + 32) >> 5) > 32) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(a.g.nmin);
    long long blocks = (a.count + kWarpsPerCta - 1) / kWarpsPerCta;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    cudaError_t e = cudaSuccess;
#define PCT_ROWS(CM)                                                                                       \
    e = cudaFuncSetAttribute(k_rows<CM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);          \
    if (e == cudaSuccess) k_rows<CM><<<(int)blocks, kThreads, smem, stream>>>(a)
    PCT_FOR_CMAX(a.g.nmin, PCT_ROWS);
#undef PCT_ROWS
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace pct
