// pct_kernels.cu -- CUDA kernels of the pCT hot path for sm_100a.
//
//   k_drop_block  fused: history stream -> hull -> MLP -> voxel walk -> a_i.x, ||a_i||^2, residual
//                 -> scatter of (r_i a_ij, 1) into the block accumulator (R12).
//                 One WARP walks one history; lane l owns the CONTIGUOUS chunk of segments
//                 [l*C, (l+1)*C), C = ceil((K+1)/32) (the MLP node at depth k*h is closed-form in
//                 k, there is no recurrence along the path) and walks it in a rolled loop, merging
//                 runs of equal voxels and summing ||a_i||^2 as it goes; the at most 31 lane seams
//                 are patched with three shuffles.  The row (voxel, length, run-head flag) goes to a
//                 per-warp buffer in SHARED memory and is read back segment-major (lane l takes
//                 segments 32 i + l) by the gather pass (a_i.x) and the scatter pass, so that
//                 neighbouring lanes touch neighbouring voxels and their L2 requests coalesce.  The
//                 path is computed once per sweep and never touches global memory.
//   k_update      x_j += lambda * Delta_j / max(1, c_j); accumulator zeroed; DROP block index advanced.
//   k_rows        inspection: the same walk, rows written out instead of consumed.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "pct_walk.cuh"
#include "pct_walk16.cuh"

namespace pct {

size_t drop_smem_bytes(int nmin) { return (size_t)smem_layout(nmin).total; }

// (checking build only) print and clear the violation counters of the block engine's kernels
void bounds_dump(const char* tag) {
#ifdef PCT_CHECK_BOUNDS
    bounds_dump_tu(tag);
#else
    (void)tag;
#endif
}

static int sm_count() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        (void)cudaGetLastError();
        return 148;
    }
    return sms;
}

// Work queue of one DROP block.  Phase 0 is STATIC: warp w of the grid owns item w (about half of
// its fair share of the block, at most kBatch histories) without touching the ticket counter, so
// the launch does not open with every warp hitting one address.  The rest is guided
// self-scheduling over one atomic ticket counter: items of half, a quarter, ... of the static size,
// each phase covering half of what is left, down to single histories -- a warp that draws one of
// the last big items stays busy for that many walks, so the work behind it must be fine-grained
// enough for the other warps to fill that time.  Small blocks get smaller items so that they still
// spread over the whole grid.
#ifndef PCT_QUEUE_HEAD_SHIFT
#define PCT_QUEUE_HEAD_SHIFT 2  // dynamic phase 1 covers left - (left >> shift) histories
#endif
#ifndef PCT_QUEUE_DIV
#define PCT_QUEUE_DIV 2  // static items: 1/DIV of a warp's fair share of the block
#endif
#ifndef PCT_QUEUE_PHASES
#define PCT_QUEUE_PHASES 4
#endif
constexpr int kPhases = PCT_QUEUE_PHASES;
struct Queue {
    long long first, count;
    int size[kPhases];                  // histories per item
    unsigned long long item0[kPhases];  // first ticket of the phase
    long long hist0[kPhases];           // first history of the phase (relative to `first`)
    unsigned long long n_static;        // tickets [0, n_static) are owned by warps, not drawn
    unsigned long long n_items;
    bool interleave;                    // static items strided by n_static (ordered blocks)
};

__device__ __forceinline__ Queue make_queue(long long first, long long count, long long n_warps) {
    Queue q;
    q.first = first;
    q.count = count;
    long long big = count / (PCT_QUEUE_DIV * n_warps);
    big = big < 1 ? 1 : (big > kBatch ? kBatch : big);
    long long done = 0;
    unsigned long long items = 0;
#pragma unroll
    for (int p = 0; p < kPhases; ++p) {
        long long sz = big >> p;
        sz = sz < 1 ? 1 : sz;
        const long long left = count - done;
        long long n;
        if (p == 0) {
            n = left / sz < n_warps ? left / sz : n_warps;  // one static item per warp
        } else if (p == kPhases - 1) {
            n = (left + sz - 1) / sz;  // the last phase takes the ragged end
        } else {
            n = (left - (left >> (p == 1 ? PCT_QUEUE_HEAD_SHIFT : 1))) / sz;
        }
        q.size[p] = (int)sz;
        q.item0[p] = items;
        q.hist0[p] = done;
        items += (unsigned long long)n;
        done += n * sz;
        if (done > count) done = count;
        if (p == 0) q.n_static = (unsigned long long)n;
    }
    q.n_items = items;
    return q;
}

// Item w: histories rel0, rel0 + stride, ... (cnt of them), positions in the block's processing order.
// With the histories of a block ordered by depth slab (k_order_blocks) the static items are INTERLEAVED
// (item w takes positions w, w + n_static, w + 2 n_static, ...), so that all warps move through the order
// together and the grid works on one slab of the image at a time.  All other items are contiguous.
__device__ __forceinline__ void queue_item(const Queue& q, unsigned long long w, long long& rel0, int& cnt, long long& stride) {
    int p = 0;
#pragma unroll
    for (int t = 1; t < kPhases; ++t) p = w >= q.item0[t] ? t : p;
    if (p == 0 && q.interleave) {
        rel0 = (long long)w;
        stride = (long long)q.n_static;
        cnt = q.size[0];
        return;
    }
    const long long rel = q.hist0[p] + (long long)(w - q.item0[p]) * q.size[p];
    rel0 = rel;
    stride = 1;
    const long long left = q.count - rel;
    cnt = left < q.size[p] ? (int)left : q.size[p];
}

template <bool SPLINE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) k_drop_block(const DropArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const SmemLayout lay = smem_layout(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * lay.row_slots;
    __shared__ Queue q;  // one copy per CTA: the phase of a ticket is looked up by index
    // Programmatic dependent launch: this grid may start while the update kernel of the previous block is still
    // running (its CTAs take the SM slots the update's CTAs leave).  The table does not depend on it; everything
    // else -- the block index in ctrl, the image -- is read after the wait below, i.e. after that grid has completed
    // and its writes are visible.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the update kernel may take the slots this grid's CTAs leave
    stage_table(s_tab, a.tab, g.kmax);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (threadIdx.x == 0) {
        long long first = a.first, count = a.count;
        if (first < 0) {
            first = a.ctrl->block * a.block_size;
            count = a.n - first < a.block_size ? a.n - first : a.block_size;
        }
        q = make_queue(first, count, (long long)gridDim.x * kWarpsPerCta);
        q.interleave = a.first < 0 && a.order != nullptr;
    }
    __syncthreads();  // q is visible
    unsigned long long rows = 0, nnz_total = 0, segs = 0;
    const EmitPtrs no_emit{nullptr, nullptr, nullptr, nullptr};

    const unsigned long long gw = (unsigned long long)blockIdx.x * kWarpsPerCta + warp;
    for (bool first_item = true;; first_item = false) {
        unsigned long long w = gw;
        if (!first_item || gw >= q.n_static) {  // warp-uniform
            if (lane == 0) w = q.n_static + atomicAdd(&a.ctrl->work, 1ULL);
            w = __shfl_sync(0xffffffffu, w, 0);
        }
        if (w >= q.n_items) break;
        long long rel0, stride;
        int cnt;
        queue_item(q, w, rel0, cnt, stride);
        if (lane < cnt) {
            long long r = rel0 + lane * stride;  // position in the processing order of the block
            if (q.interleave) r = (long long)__ldg(a.order + q.first + r);  // ordered block (k_order_blocks)
            PCT_BOUND(3, q.first + r >= 0 && q.first + r < a.n);
            const Hist hh = load_history(a.H, q.first + r);
            setup_history(g, hh, s_state[lane]);
        }
        __syncwarp();
        for (int p = 0; p < cnt; ++p) {
            const PathState& S = s_state[p];
            const int K = S.K;
            if (K < 0) continue;  // skipped history: empty row (R7)
            float nrm;
            int nnz;
            walk_history<false, SPLINE>(g, S, s_tab, lane, row, nrm, nnz, no_emit);
            const int C = (K + 32) >> 5;
            float dot = gather_row(row, lane, C, a.x);
            dot = warp_sum(dot);
            nrm = warp_sum(nrm);
            if (nrm > 0.0f) {  // non-empty row (R13)
                const float r = __fdiv_rn(S.wepl - dot, nrm);
                scatter_row(row, lane, C, a.acc, r);
                rows += (lane == 0);
                nnz_total += nnz;
            }
            __syncwarp();  // the row buffer is reused by the next history
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

// ---- two histories per warp (pct_walk16.cuh) --------------------------------------------------------------------
// Shared memory: Sigma1^-1 table | PathState[warps][kBatch] | TWO row buffers per warp.
__host__ __device__ inline SmemLayout smem_layout_pair(int kmax) {
    SmemLayout l = smem_layout(kmax);
    l.row_slots = row16_slots(kmax);
    l.total = l.row_off + kWarpsPerCta * 2 * l.row_slots * (int)sizeof(float2);
    return l;
}
size_t drop_pair_smem_bytes(int kmax) { return (size_t)smem_layout_pair(kmax).total; }

// k_drop_block with the histories of an item walked two at a time, sixteen lanes each.  The item's histories are
// sorted by their node count inside the warp first (a ten-step bitonic network on the keys the set-up lanes hold), so that
// the two of a pair are about equally long: they share one chunk size.  Work queue, set-up, dependent launch and the
// counters are those of k_drop_block.
template <bool SPLINE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) k_drop_pair(const DropArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int hl = lane & 15, half = lane >> 4;
    const SmemLayout lay = smem_layout_pair(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + (warp * 2 + half) * lay.row_slots;  // this half's row buffer
    __shared__ Queue q;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    stage_table(s_tab, a.tab, g.kmax);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (threadIdx.x == 0) {
        long long first = a.first, count = a.count;
        if (first < 0) {
            first = a.ctrl->block * a.block_size;
            count = a.n - first < a.block_size ? a.n - first : a.block_size;
        }
        q = make_queue(first, count, (long long)gridDim.x * kWarpsPerCta);
        q.interleave = a.first < 0 && a.order != nullptr;
    }
    __syncthreads();
    unsigned long long rows = 0, nnz_total = 0, segs = 0;

    const unsigned long long gw = (unsigned long long)blockIdx.x * kWarpsPerCta + warp;
    for (bool first_item = true;; first_item = false) {
        unsigned long long w = gw;
        if (!first_item || gw >= q.n_static) {
            if (lane == 0) w = q.n_static + atomicAdd(&a.ctrl->work, 1ULL);
            w = __shfl_sync(0xffffffffu, w, 0);
        }
        if (w >= q.n_items) break;
        long long rel0, stride;
        int cnt;
        queue_item(q, w, rel0, cnt, stride);
        int myK = -1;
        if (lane < cnt) {
            long long r = rel0 + lane * stride;
            if (q.interleave) r = (long long)__ldg(a.order + q.first + r);
            PCT_BOUND(3, q.first + r >= 0 && q.first + r < a.n);
            const Hist hh = load_history(a.H, q.first + r);
            setup_history(g, hh, s_state[lane]);
            myK = s_state[lane].K;
        }
        __syncwarp();
        // the item's histories by node count (lanes 0-15 hold one each; kBatch <= 16): key = (K + 1) * 16 + slot, skipped
        // histories and empty slots (K = -1) first; both halves sort the same keys
        int key = __shfl_sync(0xffffffffu, myK, hl);
        key = ((key + 1) << 4) | hl;
        key = sort16(key, hl);
        for (int p = 15; p >= 1; p -= 2) {  // pairs (p, p - 1) of the sorted order, longest first
            const int ka = __shfl_sync(0xffffffffu, key, p), kb = __shfl_sync(0xffffffffu, key, p - 1);
            const int Ka = (ka >> 4) - 1, Kb = (kb >> 4) - 1;  // Ka >= Kb
            if (Ka < 0) break;                                  // nothing but skipped histories left
            if (Kb < 0) {
                // a history without a partner (odd item, or the partner was skipped): the whole warp walks it, 32 lanes,
                // in the two row buffers taken as one
                const PathState& S = s_state[ka & 15];
                float2* row32 = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * 2 * lay.row_slots;
                float nrm;
                int nnz;
                const EmitPtrs no_emit{nullptr, nullptr, nullptr, nullptr};
                walk_history<false, SPLINE>(g, S, s_tab, lane, row32, nrm, nnz, no_emit);
                const int C = (Ka + 32) >> 5;
                float dot = gather_row(row32, lane, C, a.x);
                dot = warp_sum(dot);
                nrm = warp_sum(nrm);
                if (nrm > 0.0f) {
                    const float r = __fdiv_rn(S.wepl - dot, nrm);
                    scatter_row(row32, lane, C, a.acc, r);
                    rows += (lane == 0);
                    nnz_total += nnz;
                }
                if (lane == 0) segs += Ka + 1;
                __syncwarp();
                break;  // (everything below it in the sorted order is skipped)
            }
            const PathState& S = s_state[(half == 0 ? ka : kb) & 15];
            const int C = (Ka + 16) >> 4;                       // chunk size of the pair: ceil((Ka + 1) / 16)
            float nrm;
            int nnz;
            walk_history16<SPLINE>(g, S, s_tab, hl, C, row, nrm, nnz);
            float dot = gather16_row(row, hl, C, a.x);
            dot = half_sum(dot);
            nrm = half_sum(nrm);
            const bool live = nrm > 0.0f;                       // non-empty row (R13)
            const float r = live ? __fdiv_rn(S.wepl - dot, nrm) : 0.0f;
            scatter16_row(row, hl, C, a.acc, r, live);
            if (hl == 0 && live) ++rows;
            if (live) nnz_total += nnz;
            if (hl == 0) segs += S.K + 1;
            __syncwarp();  // the row buffers are reused by the next pair
        }
        __syncwarp();  // the state records are reused by the next item
    }
    nnz_total = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)nnz_total);
    rows = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)rows);
    segs = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)segs);
    if (lane == 0) {
        atomicAdd(&a.ctrl->cur[0], rows);
        atomicAdd(&a.ctrl->cur[1], nnz_total);
        atomicAdd(&a.ctrl->cur[2], segs);
    }
}

// The pair kernel is used where two of its CTAs fit the shared memory of an SM like k_drop_block's do (not with the
// half-voxel step on wide grids, nor on grids wider than about 420 voxels: two row buffers per warp).  Building with
// -DPCT_PAIR=0 selects the one-history-per-warp kernel (k_drop_block) everywhere (the A/B build of DESIGN.md).
#ifndef PCT_PAIR
#define PCT_PAIR 1
#endif
bool pair_enabled(int kmax) { return PCT_PAIR == 1 && 2 * (drop_pair_smem_bytes(kmax) + 1024) <= 227 * 1024; }

cudaError_t drop_configure(int nmin, int* grid_out) {
    if (((nmin + 32) >> 5) > 64) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(nmin);
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_drop_block<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_drop_block<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    // the pair kernel's two row buffers per warp outgrow the 227 KB opt-in limit on wide grids (kmax above about 850): it is
    // configured, and its occupancy taken, only where it will run; elsewhere k_drop_block alone serves
    const size_t smem2 = drop_pair_smem_bytes(nmin);
    const bool pair = pair_enabled(nmin);
    if (pair && e == cudaSuccess) e = cudaFuncSetAttribute(k_drop_pair<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
    if (pair && e == cudaSuccess) e = cudaFuncSetAttribute(k_drop_pair<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
    if (e == cudaSuccess)
        e = pair ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_drop_pair<false>, kThreads, smem2)
                 : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_drop_block<false>, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *grid_out = sms * per_sm;  // persistent: every CTA slot of the chip, work handed out dynamically
    return cudaSuccess;
}

// Launch with the programmatic-stream-serialization attribute: the grid may be scheduled as soon as the previous
// kernel in the stream lets its SM slots go; the kernel itself waits (griddepcontrol.wait) before it reads anything
// the previous kernel writes.  A build with -DPCT_PDL=0 launches the plain way.
#ifndef PCT_PDL
#define PCT_PDL 1
#endif

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = PCT_PDL ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

cudaError_t launch_drop_block(const DropArgs& a, int grid, cudaStream_t stream) {
    if (a.scratch != nullptr) return launch_drop_exact(a, grid, stream);  // exact-traversal mode (pct_exact.cu)
    // never more warps than histories (small blocks: one history per warp)
    const long long cnt = a.first < 0 ? a.block_size : a.count;
    const long long need = (cnt + kWarpsPerCta - 1) / kWarpsPerCta;
    if (need < grid) grid = need < 1 ? 1 : (int)need;
    // two histories per warp pay when a warp's items hold pairs: with fewer than four histories per warp in the block
    // (items of one history) the one-history kernel is the faster one
    // a block with two to four histories per warp of the full grid runs on fewer CTAs, so that every warp gets pairs
    // (configs[1], 1e4 histories: 250 CTAs instead of 296, 30.4 -> 28.3 us per block)
    if (pair_enabled(a.g.kmax) && cnt < 4LL * grid * kWarpsPerCta && cnt >= 2LL * grid * kWarpsPerCta) {
        grid = (int)(cnt / (4LL * kWarpsPerCta));
        if (grid < 1) grid = 1;
    }
    if (pair_enabled(a.g.kmax) && cnt >= 4LL * grid * kWarpsPerCta) {
        const size_t smem2 = drop_pair_smem_bytes(a.g.kmax);
        cudaError_t e2 = a.g.path_model == 1 ? launch_pdl(k_drop_pair<true>, dim3(grid), dim3(kThreads), smem2, stream, a)
                                             : launch_pdl(k_drop_pair<false>, dim3(grid), dim3(kThreads), smem2, stream, a);
        return e2 != cudaSuccess ? e2 : cudaGetLastError();
    }
    const size_t smem = drop_smem_bytes(a.g.kmax);
    cudaError_t e = a.g.path_model == 1 ? launch_pdl(k_drop_block<true>, dim3(grid), dim3(kThreads), smem, stream, a)
                                        : launch_pdl(k_drop_block<false>, dim3(grid), dim3(kThreads), smem, stream, a);
    return e != cudaSuccess ? e : cudaGetLastError();
}

// x_j += lambda * Delta_j / max(1, c_j) (R12); c_j >= 1 wherever anything was accumulated.
__device__ __forceinline__ float updated(float xv, float2 dc, float lambda) {
    return dc.y > 0.0f ? xv + __fdiv_rn(lambda * dc.x, dc.y) : xv;
}

#ifndef PCT_UPD_UNROLL
#define PCT_UPD_UNROLL 2  // groups of four voxels a thread has in flight at once
#endif
#ifndef PCT_UPD_CTAS
#define PCT_UPD_CTAS 8  // CTAs of 256 threads per SM
#endif

__device__ __forceinline__ float4 ld4_hint(const float4* p, unsigned long long pol) {
    float4 v;
    asm volatile("ld.global.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void st4_hint(float4* p, float4 v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}

// One group = four consecutive voxels: two 128-bit accumulator loads, one 128-bit image load.  A
// thread issues the loads of PCT_UPD_UNROLL groups (a CTA-stride apart, so that every load is
// coalesced) before it touches any of them: the kernel is bound by L2 latency x bytes in flight.
// top_down: sweep the image from the last slice to the first.  With the histories of a block taken depth slab by
// depth slab (k_order_blocks) the accumulate kernel ends on the last slabs and the next one starts on the first: the
// update then finds the end of image and accumulator still in the L2 and leaves their beginning there.
__global__ void __launch_bounds__(256) k_update(float* __restrict__ x, float2* __restrict__ acc, long long n_voxels,
                                                float lambda, Ctrl* ctrl, long long n_blocks, bool top_down) {
    constexpr int UN = PCT_UPD_UNROLL;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");  // (launched while the accumulate kernel of the block drains: see launch_pdl)
    const unsigned long long keep = policy_evict_last();
#if PCT_ACC_EVICT_FIRST
    const unsigned long long stream_pol = policy_evict_first();
#define PCT_LD_ACC(p) ld4_hint(p, stream_pol)
#else
#define PCT_LD_ACC(p) (*(p))
#endif
    const long long n4 = n_voxels >> 2;
    const long long stride = (long long)gridDim.x * blockDim.x;
    float4* x4 = reinterpret_cast<float4*>(x);
    float4* a4 = reinterpret_cast<float4*>(acc);
    for (long long q0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; q0 < n4; q0 += stride * UN) {
        float4 a01[UN], a23[UN], xv[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            long long q = q0 + u * stride;
            if (q < n4) {
                if (top_down) q = n4 - 1 - q;
                a01[u] = PCT_LD_ACC(a4 + 2 * q);
                a23[u] = PCT_LD_ACC(a4 + 2 * q + 1);
                xv[u] = ld4_hint(x4 + q, keep);
            } else {
                a01[u] = a23[u] = xv[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            long long q = q0 + u * stride;
            if (top_down) q = n4 - 1 - q;
            const bool hit01 = a01[u].y > 0.0f || a01[u].w > 0.0f, hit23 = a23[u].y > 0.0f || a23[u].w > 0.0f;
            if (hit01 || hit23) {  // (q < n4 is implied: out-of-range groups were loaded as zeros)
                float4 v = xv[u];
                v.x = updated(v.x, make_float2(a01[u].x, a01[u].y), lambda);
                v.y = updated(v.y, make_float2(a01[u].z, a01[u].w), lambda);
                v.z = updated(v.z, make_float2(a23[u].x, a23[u].y), lambda);
                v.w = updated(v.w, make_float2(a23[u].z, a23[u].w), lambda);
                st4_hint(x4 + q, v, keep);
                const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                if (hit01) a4[2 * q] = z;  // (hinting these stores, or the reductions, measured no better)
                if (hit23) a4[2 * q + 1] = z;
            }
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
                          bool top_down, cudaStream_t stream) {
    const long long n4 = n_voxels >> 2;
    long long blocks = (n4 + 256 * PCT_UPD_UNROLL - 1) / (256 * PCT_UPD_UNROLL);
    if (blocks < 1) blocks = 1;
    const long long cap = (long long)sm_count() * PCT_UPD_CTAS;
    if (blocks > cap) blocks = cap;
    const cudaError_t e = launch_pdl(k_update, dim3((int)blocks), dim3(256), 0, stream, x, acc, n_voxels, lambda, ctrl, n_blocks, top_down);
    return e != cudaSuccess ? e : cudaGetLastError();
}

// inspection: de-interleave the accumulator into Delta and c (in the voxel order of include/pct.h), and zero it
__global__ void k_split_acc(float2* __restrict__ acc, float* __restrict__ delta, float* __restrict__ cnt, Geom g) {
    const long long n = (long long)g.nx * g.ny * g.nz;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const int i = (int)(v % g.nx), j = (int)((v / g.nx) % g.ny), k = (int)(v / ((long long)g.nx * g.ny));
        const int slot = voxel_slot(i, j, k, g.nxp, g.slice_p);
        const float2 dc = acc[slot];
        delta[v] = dc.x;
        cnt[v] = dc.y;
        acc[slot] = make_float2(0.f, 0.f);
    }
}

cudaError_t launch_split_acc(float2* acc, float* delta, float* cnt, const Geom& g, cudaStream_t stream) {
    const long long n = (long long)g.nx * g.ny * g.nz;
    long long blocks = (n + 255) / 256;
    const long long cap = (long long)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    k_split_acc<<<(int)blocks, 256, 0, stream>>>(acc, delta, cnt, g);
    return cudaGetLastError();
}

// Image I/O: the caller's order i + nx (j + ny k) <-> the storage order (voxel_slot).  to_storage: ext -> x, else x -> ext.
__global__ void k_image_io(float* __restrict__ x, float* __restrict__ ext, Geom g, bool to_storage) {
    const long long n = (long long)g.nx * g.ny * g.nz;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const int i = (int)(v % g.nx), j = (int)((v / g.nx) % g.ny), k = (int)(v / ((long long)g.nx * g.ny));
        const int slot = voxel_slot(i, j, k, g.nxp, g.slice_p);
        if (to_storage)
            x[slot] = ext[v];
        else
            ext[v] = x[slot];
    }
}

cudaError_t launch_image_io(float* x, float* ext, const Geom& g, bool to_storage, cudaStream_t stream) {
    const long long n = (long long)g.nx * g.ny * g.nz;
    long long blocks = (n + 255) / 256;
    const long long cap = (long long)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    k_image_io<<<(int)blocks, 256, 0, stream>>>(x, ext, g, to_storage);
    return cudaGetLastError();
}

// inspection: one warp per history, rows written out (include/pct.h, pct_debug_rows).  The walk,
// the run heads and the non-zero count are those of the hot path; only the merged length of a
// run (which the hot path never forms: it needs ||a_i||^2 and the unmerged scatter only) is
// summed here, from the segment lengths just written.
template <bool SPLINE>
__global__ void __launch_bounds__(kThreads) k_rows(const RowsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const SmemLayout lay = smem_layout(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * lay.row_slots;
    stage_table(s_tab, a.tab, g.kmax);
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
            float nrm;
            int nnz;
            walk_history<true, SPLINE>(g, S, s_tab, lane, row, nrm, nnz, em);
            nnz_total = __reduce_add_sync(0xffffffffu, nnz);
            // the row as the hot path sees it: read back from the row buffer, segment-major
            for (int k = lane; k <= K; k += 32) {
                const float2 e = row[row_slot(k)];
                if (em.seg_idx) {  // reported as the linear index i + nx (j + ny k) of include/pct.h, not as the storage slot
                    int lin = __float_as_int(e.x);
                    if (lin >= 0) {
                        int vi, vj, vk;
                        voxel_of_slot(lin, g.nxp, g.slice_p, vi, vj, vk);
                        lin = vi + g.nx * (vj + g.ny * vk);
                    }
                    em.seg_idx[k] = lin;
                }
                if (em.seg_len && __float_as_int(e.x) >= 0) em.seg_len[k] = fabsf(e.y);
                if (em.row_len) em.row_len[k] = __float_as_int(e.y) < 0 ? 1.0f : 0.0f;
            }
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

// inspection of the two-histories-per-warp walk (pct_walk16.cuh; pct_set_option PCT_OPT_ROWS_PAIR): histories (2 w, 2 w + 1) of the range
// are walked side by side exactly as k_drop_pair walks a pair, and the rows are read back from the two row buffers.
// Node positions are not written by this walk (they are k_rows's, the same node_pair code).
template <bool SPLINE>
__global__ void __launch_bounds__(kThreads) k_rows_pair(const RowsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int hl = lane & 15, half = lane >> 4;
    const SmemLayout lay = smem_layout_pair(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + (warp * 2 + half) * lay.row_slots;
    stage_table(s_tab, a.tab, g.kmax);
    const long long n_pairs = (a.count + 1) / 2;
    for (long long pr = (long long)blockIdx.x * kWarpsPerCta + warp; pr < n_pairs; pr += (long long)gridDim.x * kWarpsPerCta) {
        const long long r = 2 * pr + half;  // this half's history
        const bool have = r < a.count;
        if (hl == 0) {
            s_state[half].K = -1;
            if (have) {
                const Hist hh = load_history(a.H, a.first + r);
                setup_history(g, hh, s_state[half]);
            }
        }
        __syncwarp();
        const int Ka = s_state[0].K, Kb = s_state[1].K;
        const int Kmax = Ka > Kb ? Ka : Kb;
        int nnz_total = 0;
        const int K = s_state[half].K;
        if (Kmax >= 0) {
            const PathState& S = s_state[K >= 0 ? half : (half ^ 1)];  // (a half without a path walks its partner's, muted)
            const int C = (Kmax + 16) >> 4;
            float nrm;
            int nnz;
            walk_history16<SPLINE>(g, S, s_tab, hl, C, row, nrm, nnz);
            nnz_total = nnz;
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) nnz_total += __shfl_xor_sync(0xffffffffu, nnz_total, o, 16);
            if (have && K >= 0) {
                int32_t* o_idx = a.seg_idx ? a.seg_idx + (size_t)r * a.max_seg : nullptr;
                float* o_len = a.seg_len ? a.seg_len + (size_t)r * a.max_seg : nullptr;
                float* o_row = a.row_len ? a.row_len + (size_t)r * a.max_seg : nullptr;
                for (int k = hl; k <= K; k += 16) {
                    const float2 e = row[row_slot(k)];
                    int lin = __float_as_int(e.x);
                    if (lin >= 0) {
                        int vi, vj, vk;
                        voxel_of_slot(lin, g.nxp, g.slice_p, vi, vj, vk);
                        lin = vi + g.nx * (vj + g.ny * vk);
                    }
                    if (o_idx) o_idx[k] = lin;
                    if (o_len) o_len[k] = fabsf(e.y);
                    if (o_row) o_row[k] = __float_as_int(e.y) < 0 ? 1.0f : 0.0f;
                }
            }
            __syncwarp();
            if (have && K >= 0 && a.row_len && a.seg_idx && a.seg_len) {
                int32_t* o_idx = a.seg_idx + (size_t)r * a.max_seg;
                float* o_len = a.seg_len + (size_t)r * a.max_seg;
                float* o_row = a.row_len + (size_t)r * a.max_seg;
                for (int k = hl; k <= K; k += 16) {
                    if (o_row[k] > 0.0f) {
                        const int idx = o_idx[k];
                        float lm = o_len[k];
                        for (int m = k + 1; m <= K && o_idx[m] == idx; ++m) lm += o_len[m];
                        o_row[k] = lm;
                    }
                }
            }
        }
        if (hl == 0 && have) {
            a.nseg[r] = K >= 0 ? K + 1 : 0;
            a.nnz[r] = K >= 0 ? nnz_total : 0;
        }
        __syncwarp();
    }
}

cudaError_t launch_rows(const RowsArgs& a, bool pair_walk, cudaStream_t stream) {
    if (((a.g.kmax + 32) >> 5) > 64) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(a.g.kmax);
    long long blocks = (a.count + kWarpsPerCta - 1) / kWarpsPerCta;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    cudaError_t e = cudaSuccess;
    if (pair_walk && a.nodes == nullptr && pair_enabled(a.g.kmax)) {  // the hot path's pair walk, inspected
        const size_t smem2 = drop_pair_smem_bytes(a.g.kmax);
        if (a.g.path_model == 1) {
            e = cudaFuncSetAttribute(k_rows_pair<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
            if (e == cudaSuccess) k_rows_pair<true><<<(int)blocks, kThreads, smem2, stream>>>(a);
        } else {
            e = cudaFuncSetAttribute(k_rows_pair<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
            if (e == cudaSuccess) k_rows_pair<false><<<(int)blocks, kThreads, smem2, stream>>>(a);
        }
        return e != cudaSuccess ? e : cudaGetLastError();
    }
    if (a.g.path_model == 1) {
        e = cudaFuncSetAttribute(k_rows<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) k_rows<true><<<(int)blocks, kThreads, smem, stream>>>(a);
    } else {
        e = cudaFuncSetAttribute(k_rows<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) k_rows<false><<<(int)blocks, kThreads, smem, stream>>>(a);
    }
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

// ---- processing order of the histories inside a DROP block -------------------------------------
// The block update is a sum over the rows of the block (R12), so the library may take them in any
// order (R14: never across blocks).  A path stays within a slice or two of the image (mrad slopes),
// so histories taken DEPTH SLAB by depth slab touch 1/n_slabs of image and accumulator at a time:
// the gather and the reductions hit the L2 even when image + accumulator (126 MB at 256 x 256 x 160)
// exceed it.  One counting sort per block on the slab of the straight entry ray at u = 0.  An ordering
// only: any key gives the same sums.  (A second key, longest histories first inside a slab so that the
// launch ends on short ones, was measured: no gain.)
constexpr int kOrderBins = 64;  // at most that many slabs

__device__ __forceinline__ int order_key(const HistPtrs& H, const Geom& g, int n_slabs, long long i) {
    const float vc = __ldg(H.v_in + i) - __ldg(H.dv_in + i) * g.u_in;  // straight entry ray at u = 0
    float fs = (vc + g.zmax) / (2.0f * g.zmax) * (float)n_slabs;
    fs = fs >= 0.0f ? fs : 0.0f;  // (NaN -> 0)
    return fs < (float)n_slabs ? (int)fs : n_slabs - 1;
}

__global__ void __launch_bounds__(512) k_order_blocks(const HistPtrs H, const Geom g, long long n, long long block_size,
                                                      long long first_block, long long n_blocks, int n_slabs, uint32_t* __restrict__ order) {
    __shared__ unsigned bins[kOrderBins];
    for (long long b = first_block + blockIdx.x; b < first_block + n_blocks; b += gridDim.x) {
        const long long first = b * block_size;
        const long long count = n - first < block_size ? n - first : block_size;
        for (int k = threadIdx.x; k < kOrderBins; k += blockDim.x) bins[k] = 0u;
        __syncthreads();
        for (long long r = threadIdx.x; r < count; r += blockDim.x) atomicAdd(&bins[order_key(H, g, n_slabs, first + r)], 1u);
        __syncthreads();
        if (threadIdx.x < 32) {  // exclusive scan of the bin counts by one warp
            unsigned carry = 0u;
            for (int k0 = 0; k0 < kOrderBins; k0 += 32) {
                const int k = k0 + threadIdx.x;
                const unsigned c = k < kOrderBins ? bins[k] : 0u;
                unsigned incl = c;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const unsigned up = __shfl_up_sync(0xffffffffu, incl, o);
                    if ((int)threadIdx.x >= o) incl += up;
                }
                if (k < kOrderBins) bins[k] = carry + incl - c;
                carry += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
        __syncthreads();
        for (long long r = threadIdx.x; r < count; r += blockDim.x) {
            const unsigned pos = atomicAdd(&bins[order_key(H, g, n_slabs, first + r)], 1u);
            order[first + pos] = (uint32_t)r;
        }
        __syncthreads();
    }
}

cudaError_t launch_order_blocks(const HistPtrs& H, const Geom& g, long long n, long long block_size, long long first_block,
                                long long n_blocks, int n_slabs, uint32_t* order, cudaStream_t stream) {
    if (n_blocks < 1) return cudaSuccess;
    n_slabs = n_slabs < 1 ? 1 : (n_slabs > kOrderBins ? kOrderBins : n_slabs);
    const long long cap = (long long)sm_count() * 4;
    const long long grid = n_blocks < cap ? n_blocks : cap;
    k_order_blocks<<<(int)grid, 512, 0, stream>>>(H, g, n, block_size, first_block, n_blocks, n_slabs, order);
    return cudaGetLastError();
}

// Object-frame entry point (include/pct.h pct_set_histories_xyz; R32): tracker hits (x, y, z) in the object
// frame are carried along their straight rays to the tracker planes of the rule.  fp32, this operation order:
//   u = fma(y, cos, -(x sin));  t = fma(x, cos, y sin);  t_pl = fma(theta_t, u_pl - u, t);  v_pl = fma(theta_v, u_pl - u, z)
__global__ void __launch_bounds__(256) k_xyz_to_beam(float u_pl, long long n, const float* __restrict__ x, const float* __restrict__ y,
                                                     const float* __restrict__ z, const float* __restrict__ tht, const float* __restrict__ thv,
                                                     const uint16_t* __restrict__ proj, const float* __restrict__ pcos,
                                                     const float* __restrict__ psin, int n_proj, float* __restrict__ t_out,
                                                     float* __restrict__ v_out) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        int p = (int)proj[i];
        p = p < n_proj ? p : n_proj - 1;
        const float cs = __ldg(pcos + p), sn = __ldg(psin + p);
        const float u = __fmaf_rn(y[i], cs, -__fmul_rn(x[i], sn));
        const float t = __fmaf_rn(x[i], cs, __fmul_rn(y[i], sn));
        const float du = __fsub_rn(u_pl, u);
        t_out[i] = __fmaf_rn(tht[i], du, t);
        v_out[i] = __fmaf_rn(thv[i], du, z[i]);
    }
}

cudaError_t launch_xyz_to_beam(float u_pl, long long n, const float* x, const float* y, const float* z, const float* tht, const float* thv,
                               const uint16_t* proj, const float* pcos, const float* psin, int n_proj, float* t_out, float* v_out,
                               cudaStream_t stream) {
    long long blocks = (n + 255) / 256;
    const long long cap = (long long)sm_count() * 16;
    if (blocks > cap) blocks = cap;
    k_xyz_to_beam<<<(int)blocks, 256, 0, stream>>>(u_pl, n, x, y, z, tht, thv, proj, pcos, psin, n_proj, t_out, v_out);
    return cudaGetLastError();
}

// CARP (R29): the new solution is the arithmetic mean of the P string solutions, voxel by
// voxel; summed in the order of the strings (deterministic).  xs = P images of n voxels, back to back.
// xs = P images, `pitch` voxels apart.
__global__ void __launch_bounds__(256) k_mean(float* __restrict__ x, const float* __restrict__ xs, int n_strings, long long n, long long pitch) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    const float fp = (float)n_strings;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        float s = 0.0f;
        for (int p = 0; p < n_strings; ++p) s += xs[(long long)p * pitch + j];
        x[j] = __fdiv_rn(s, fp);
    }
}


cudaError_t launch_mean(float* x, const float* xs, int n_strings, long long n, long long pitch, cudaStream_t stream) {
    long long blocks = (n + 255) / 256;
    const long long cap = (long long)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    k_mean<<<(int)blocks, 256, 0, stream>>>(x, xs, n_strings, n, pitch);
    return cudaGetLastError();
}

// pct_get_stats after CARP: the counters of the strings' last sweeps, added up into the context's.  src = the `last`
// array of string 0, the strings' control blocks `pitch` bytes apart.
// inspection: the rule's 1/a and sqrt(a) (pct_rule.cuh: hardware approximation + one FMA Newton step, no range test)
// against the IEEE intrinsics __frcp_rn / __fsqrt_rn for EVERY fp32 bit pattern in [lo, hi] -- the argument ranges the
// rule feeds them are swept in full by tests/test_gpu_parity.py.  out[0] counts the patterns whose results
// differ in any bit, out[1] keeps the lowest such pattern.
__global__ void k_rule_sweep(int which, uint32_t lo, uint32_t hi, unsigned long long* out) {
    const unsigned long long n = (unsigned long long)hi - lo + 1ULL, pairs = (n + 1ULL) >> 1;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    unsigned long long bad = 0ULL, first = ~0ULL;
    for (unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; q < pairs; q += stride) {
        const unsigned long long b0 = lo + 2ULL * q, b1 = b0 + 1ULL <= hi ? b0 + 1ULL : b0;
        const float a0 = __uint_as_float((uint32_t)b0), a1 = __uint_as_float((uint32_t)b1);
        float r0, r1;
        upk(which == 0 ? rcp_rn_normal2(pk(a0, a1)) : sqrt_rn_normal2(pk(a0, a1)), r0, r1);
        const float w0 = which == 0 ? __frcp_rn(a0) : __fsqrt_rn(a0), w1 = which == 0 ? __frcp_rn(a1) : __fsqrt_rn(a1);
        if (__float_as_uint(r0) != __float_as_uint(w0)) ++bad, first = b0 < first ? b0 : first;
        if (b1 != b0 && __float_as_uint(r1) != __float_as_uint(w1)) ++bad, first = b1 < first ? b1 : first;
    }
    if (bad) {
        atomicAdd(&out[0], bad);
        atomicMin(&out[1], first);
    }
}

cudaError_t launch_rule_sweep(int which, uint32_t lo, uint32_t hi, unsigned long long* out, cudaStream_t stream) {
    k_rule_sweep<<<sm_count() * 8, 256, 0, stream>>>(which, lo, hi, out);
    return cudaGetLastError();
}

__global__ void k_sum_stats(unsigned long long* dst, const unsigned long long* src, size_t pitch, int n_strings) {
    if (threadIdx.x < 4) {
        unsigned long long s = 0;
        for (int p = 0; p < n_strings; ++p)
            s += reinterpret_cast<const unsigned long long*>(reinterpret_cast<const char*>(src) + (size_t)p * pitch)[threadIdx.x];
        dst[threadIdx.x] = s;
    }
}

cudaError_t launch_sum_stats(unsigned long long* dst, const unsigned long long* src, size_t pitch, int n_strings, cudaStream_t stream) {
    k_sum_stats<<<1, 32, 0, stream>>>(dst, src, pitch, n_strings);
    return cudaGetLastError();
}

}  // namespace pct
