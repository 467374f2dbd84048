// pct_exact.cu -- the EXACT voxel traversal of the path polyline (R34), selected with
// pct_set_walk(ctx, PCT_WALK_EXACT).  PAPER.md:44 defines a row of A as the "path lengths in voxels touched by the
// proton"; the graded path credits every polyline segment to the voxel of its midpoint (R10), this mode cuts every
// segment A -> B at the voxel faces it crosses and credits every piece to the voxel it lies in:
//     gA = fma(A, 1/h, n/2), gB likewise, d = gB - gA                                  (grid coordinates, per axis)
//     per axis x, y, z: if floor(gA) != floor(gB): for every integer p, min + 1 <= p <= max of the two floors, ascending:
//         t = (p - gA) / d clamped to [0, 1]                                           (at most kMaxCuts cuts in all)
//     cuts sorted ascending; consecutive cuts t0 < t1 (0 and 1 included) give a piece of length (t1 - t0) * len in the
//     voxel floor(fma(0.5 (t0 + t1), d, gA)); pieces of zero length are dropped
// fp32 with explicit rounding, in exactly this operation order (R34): it decides voxel indices.
//
// A variant for accuracy studies, not the throughput path: one warp per history, lane l walks the segments
// [l C, (l+1) C) one after another, merges consecutive pieces of one voxel and writes its runs to a scratch area of the
// warp in GLOBAL memory (a lane's chunk yields a variable number of runs); the lane seams are patched as in the
// midpoint kernel; gather and scatter then go over each lane's own runs.  Nodes, hull, DROP block update and the block
// loop are those of the graded path (pct_kernels.cu).
#include "pct_walk.cuh"

namespace pct {

constexpr int kMaxCuts = 24;

__device__ __forceinline__ float3 obj3(float x, float y, float z) { return make_float3(x, y, z); }

// f(voxel slot or -1, piece length) for every piece of the segment A -> B, in order along the segment.
template <typename F>
__device__ __forceinline__ void for_each_piece(const Geom& g, const float3 A, const float3 B, F&& f) {
    const float dx = __fsub_rn(B.x, A.x), dy = __fsub_rn(B.y, A.y), dz = __fsub_rn(B.z, A.z);
    const float len = __fsqrt_rn(__fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))));
    const float a3[3] = {A.x, A.y, A.z}, b3[3] = {B.x, B.y, B.z}, half[3] = {g.hx, g.hy, g.hz};
    float ga[3], d[3], ts[kMaxCuts];
    int nt = 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        ga[c] = __fmaf_rn(a3[c], g.inv_h, half[c]);
        const float gb = __fmaf_rn(b3[c], g.inv_h, half[c]);
        d[c] = __fsub_rn(gb, ga[c]);
        const float fa = floorf(ga[c]), fb = floorf(gb);
        if (fa != fb) {
            const float lo = fa < fb ? fa : fb, hi = fa < fb ? fb : fa;
            for (float p = __fadd_rn(lo, 1.0f); p <= hi && nt < kMaxCuts; p = __fadd_rn(p, 1.0f)) {
                float t = __fdiv_rn(__fsub_rn(p, ga[c]), d[c]);
                t = t < 0.0f ? 0.0f : (t > 1.0f ? 1.0f : t);
                ts[nt++] = t;
            }
        }
    }
    for (int i = 1; i < nt; ++i) {  // insertion sort, ascending (three cuts at most on ordinary paths)
        const float v = ts[i];
        int j = i - 1;
        while (j >= 0 && ts[j] > v) {
            ts[j + 1] = ts[j];
            --j;
        }
        ts[j + 1] = v;
    }
    float t0 = 0.0f;
    for (int j = 0; j <= nt; ++j) {
        const float t1 = j < nt ? ts[j] : 1.0f;
        if (t1 > t0) {
            const float tm = __fmul_rn(0.5f, __fadd_rn(t0, t1));
            const int vox = voxel_of(g, __fmaf_rn(tm, d[0], ga[0]), __fmaf_rn(tm, d[1], ga[1]), __fmaf_rn(tm, d[2], ga[2]));
            f(vox, __fmul_rn(__fsub_rn(t1, t0), len));
            t0 = t1;
        }
    }
}

// voxel_of tests 0 <= g < n on the bit patterns and relies on g never being -0 (pct_rule.cuh).  Here g = fma(tm, d, gA)
// can round to -0 only if it is an exact zero of opposite-signed terms, which rounds to +0 in round-to-nearest: the
// same argument holds.  (A negative g has a pattern above that of n and is rejected.)

// The segments [k0, k0 + C) of the lane, one after another: f(segment index, A, B) for those that exist (<= K).
template <bool SPLINE, typename F>
__device__ __forceinline__ void for_each_segment(const Geom& g, const PathState& st, const float4* s_tabA, const float4* s_tabB, int pad_mask,
                                                 int k0, int C, int K, F&& f) {
    const float3 exitP = to_object(st, st.t2, st.u2, st.v2);
    float3 cur = k0 == 0 ? to_object(st, st.t0, st.u0, st.v0) : lo3(node_pair<SPLINE>(st, s_tabA, s_tabB, pad_mask, k0, K, exitP));
    float3 spare = cur;
    for (int s = 0; s < C && k0 + s <= K; ++s) {
        float3 nxt;
        if ((s & 1) == 0) {
            const Node2 P = node_pair<SPLINE>(st, s_tabA, s_tabB, pad_mask, k0 + s + 1, K, exitP);  // nodes k0+s+1, k0+s+2
            nxt = lo3(P);
            spare = hi3(P);
        } else {
            nxt = spare;
        }
        f(k0 + s, cur, nxt);
        cur = nxt;
    }
}

struct TabSel {
    const float4 *A, *B;
    int pad_mask;
};
__device__ __forceinline__ TabSel select_table(const Geom& g, const float4* s_tab, int C) {
    const int tab_n = tab_slots(g.kmax);
    TabSel t;
    t.pad_mask = (C & 1) ? 0 : -1;
    t.A = s_tab + ((C & 1) ? 2 * tab_n : 0);
    t.B = t.A + tab_n;
    return t;
}

template <bool SPLINE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) k_drop_exact(const DropArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const SmemLayout lay = smem_layout(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    stage_table(s_tab, a.tab, g.kmax);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    long long first = a.first, count = a.count;
    if (first < 0) {
        first = a.ctrl->block * a.block_size;
        count = a.n - first < a.block_size ? a.n - first : a.block_size;
    }
    const long long n_warps = (long long)gridDim.x * kWarpsPerCta;
    const long long gw = (long long)blockIdx.x * kWarpsPerCta + warp;
    float2* mine = a.scratch + ((size_t)gw * 32 + lane) * a.cap_lane;  // this lane's runs
    unsigned long long rows = 0, nnz_total = 0, pieces_total = 0;
    const unsigned long long pol = policy_evict_last();
    for (long long r = gw; r < count; r += n_warps) {  // (static round robin: the variant is not tuned for the tail)
        if (lane == 0) {
            const Hist hh = load_history(a.H, first + r);
            setup_history(g, hh, s_state[0]);
        }
        __syncwarp();
        const PathState st = s_state[0];
        __syncwarp();
        const int K = st.K;
        if (K < 0) continue;
        const int C = (K + 32) >> 5, k0 = lane * C;
        const TabSel tb = select_table(g, s_tab, C);
        // ---- walk: pieces -> runs of equal voxels (merged inside the lane), stored to the lane's scratch ----
        int n_runs = 0, run_idx = -2, n_fresh = 0, nnz = 0, n_pieces = 0;
        float run_len = 0.0f, first_len = 0.0f, nrm = 0.0f;
        bool overflow = false;
        auto flush = [&]() {  // the finished run goes to the scratch (outside runs too: they break a run across lanes)
            if (n_runs < a.cap_lane)
                mine[n_runs] = make_float2(__int_as_float(run_idx), run_len);
            else
                overflow = true;
            ++n_runs;
        };
        for_each_segment<SPLINE>(g, st, tb.A, tb.B, tb.pad_mask, k0, C, K, [&](int, const float3 A, const float3 B) {
            for_each_piece(g, A, B, [&](int vox, float plen) {
                ++n_pieces;
                if (vox != run_idx) {
                    if (n_fresh > 0) {
                        nrm = __fmaf_rn(run_len, run_len, nrm);
                        if (n_fresh == 1) first_len = run_len;
                        flush();
                    }
                    ++n_fresh;
                    run_idx = vox;
                    run_len = plen;
                    nnz += vox >= 0 ? 1 : 0;
                } else {
                    run_len += plen;
                }
            });
        });
        if (n_fresh > 0) {
            nrm = __fmaf_rn(run_len, run_len, nrm);
            if (n_fresh == 1) first_len = run_len;
            flush();
        }
        // (the squared lengths of runs OUTSIDE the grid must not count)
        // -> recomputed below from the stored runs, which also applies the seam corrections
        const bool whole = n_fresh == 1;
        const int last_idx = n_fresh > 0 ? run_idx : -3;  // (-3: the lane has no piece at all: nothing to continue)
        const float last_len = run_len;
        // ---- lane seams: the lane's first run may continue the last run of the nearest earlier lane that has pieces ----
        // Lanes past the end of the path have no pieces; they sit at the high lanes only (chunks are contiguous), so
        // the previous lane always has pieces when this one has.
        const int lin0 = n_fresh > 0 ? __float_as_int(mine[0].x) : -1;
        const int prev_idx = __shfl_up_sync(0xffffffffu, last_idx, 1);
        const float prev_len = __shfl_up_sync(0xffffffffu, last_len, 1);
        const bool prev_whole = __shfl_up_sync(0xffffffffu, (int)whole, 1) != 0;
        const bool cont = lane > 0 && n_fresh > 0 && lin0 >= 0 && lin0 == prev_idx;
        const float base = cont ? prev_len : 0.0f;
        float carry = base;
        if (__any_sync(0xffffffffu, cont && prev_whole)) {
            for (int it = 0; it < 31; ++it) {
                const float up = __shfl_up_sync(0xffffffffu, carry, 1);
                const float nc = (cont && prev_whole) ? base + up : base;
                const bool changed = nc != carry;
                carry = nc;
                if (!__any_sync(0xffffffffu, changed)) break;
            }
        }
        // ||a||^2 over the runs inside the grid, with (q + p)^2 = q^2 + 2 q p + p^2 at the seams
        const int stored = n_runs < a.cap_lane ? n_runs : a.cap_lane;
        float nr = 0.0f, dot = 0.0f;
        for (int j = 0; j < stored; ++j) {
            const float2 e = mine[j];
            const int vox = __float_as_int(e.x);
            if (vox >= 0) {
                nr = __fmaf_rn(e.y, e.y, nr);
                dot = __fmaf_rn(e.y, ld_image(a.x + vox, pol), dot);
            }
        }
        if (cont) {
            nr = __fmaf_rn(2.0f * carry, first_len, nr);
            --nnz;
        }
        (void)nrm;
        dot = warp_sum(dot);
        nr = warp_sum(nr);
        if (__any_sync(0xffffffffu, overflow)) {  // more runs than the scratch holds (slopes far beyond any tracker's): flagged
            if (lane == 0) atomicAdd(&a.ctrl->cur[3], 1ULL);
            continue;
        }
        if (nr > 0.0f) {
            const float rr = __fdiv_rn(st.wepl - dot, nr);
            for (int j = 0; j < stored; ++j) {
                const float2 e = mine[j];
                red_add_v2(a.acc, __float_as_int(e.x), rr * e.y, (j == 0 && cont) ? 0.0f : 1.0f);
            }
            rows += (lane == 0);
            nnz_total += nnz;
        }
        pieces_total += n_pieces;
    }
    nnz_total = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)nnz_total);
    pieces_total = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)pieces_total);
    if (lane == 0) {
        atomicAdd(&a.ctrl->cur[0], rows);
        atomicAdd(&a.ctrl->cur[1], nnz_total);
        atomicAdd(&a.ctrl->cur[2], pieces_total);
    }
}

// inspection: the pieces of histories [first, first + count) written out (pct_debug_rows in the exact mode): nseg = number
// of pieces, seg_idx / seg_len per piece, row_len = merged length at the first piece of every run, nodes as always.
template <bool SPLINE>
__global__ void __launch_bounds__(kThreads) k_rows_exact(const RowsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const SmemLayout lay = smem_layout(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    stage_table(s_tab, a.tab, g.kmax);
    for (long long r = (long long)blockIdx.x * kWarpsPerCta + warp; r < a.count; r += (long long)gridDim.x * kWarpsPerCta) {
        if (lane == 0) {
            const Hist hh = load_history(a.H, a.first + r);
            setup_history(g, hh, s_state[0]);
        }
        __syncwarp();
        const PathState st = s_state[0];
        __syncwarp();
        const int K = st.K;
        int n_total = 0, nnz_total = 0;
        if (K >= 0) {
            int32_t* o_idx = a.seg_idx ? a.seg_idx + (size_t)r * a.max_seg : nullptr;
            float* o_len = a.seg_len ? a.seg_len + (size_t)r * a.max_seg : nullptr;
            float* o_row = a.row_len ? a.row_len + (size_t)r * a.max_seg : nullptr;
            float* o_nodes = a.nodes ? a.nodes + (size_t)r * (a.max_seg + 1) * 3 : nullptr;
            const int C = (K + 32) >> 5, k0 = lane * C;
            const TabSel tb = select_table(g, s_tab, C);
            int mine = 0;  // pass 1: how many pieces this lane has
            for_each_segment<SPLINE>(g, st, tb.A, tb.B, tb.pad_mask, k0, C, K, [&](int, const float3 A, const float3 B) {
                for_each_piece(g, A, B, [&](int, float) { ++mine; });
            });
            int incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += up;
            }
            n_total = __shfl_sync(0xffffffffu, incl, 31);
            int pos = incl - mine;  // pass 2: the pieces at their place in the history's list
            for_each_segment<SPLINE>(g, st, tb.A, tb.B, tb.pad_mask, k0, C, K, [&](int seg, const float3 A, const float3 B) {
                if (o_nodes) {
                    o_nodes[3 * seg + 0] = A.x; o_nodes[3 * seg + 1] = A.y; o_nodes[3 * seg + 2] = A.z;
                    if (seg == K) { o_nodes[3 * (K + 1) + 0] = B.x; o_nodes[3 * (K + 1) + 1] = B.y; o_nodes[3 * (K + 1) + 2] = B.z; }
                }
                for_each_piece(g, A, B, [&](int vox, float plen) {
                    if (pos < a.max_seg) {
                        if (o_idx) {
                            int lin = vox;
                            if (lin >= 0) {
                                int vi, vj, vk;
                                voxel_of_slot(lin, g.nxp, g.slice_p, vi, vj, vk);
                                lin = vi + g.nx * (vj + g.ny * vk);
                            }
                            o_idx[pos] = lin;
                        }
                        if (o_len) o_len[pos] = plen;
                    }
                    ++pos;
                });
            });
            __syncwarp();
            __threadfence_block();
            // run heads and merged lengths, from the list just written
            const int n_out = n_total < a.max_seg ? n_total : a.max_seg;
            int heads = 0;
            if (o_idx && o_len) {
                for (int k = lane; k < n_out; k += 32) {
                    const int idx = o_idx[k];
                    const bool head = idx >= 0 && (k == 0 || o_idx[k - 1] != idx);
                    float lm = 0.0f;
                    if (head) {
                        ++heads;
                        lm = o_len[k];
                        for (int m = k + 1; m < n_out && o_idx[m] == idx; ++m) lm += o_len[m];
                    }
                    if (o_row) o_row[k] = lm;
                }
            }
            nnz_total = __reduce_add_sync(0xffffffffu, heads);
        }
        if (lane == 0) {
            a.nseg[r] = n_total;
            a.nnz[r] = nnz_total;
        }
        __syncwarp();
    }
}

size_t exact_scratch_bytes(int kmax, int grid, int* cap_lane_out) {
    const int cmax = (kmax + 32) >> 5;
    const int cap = 8 * cmax + 8;  // runs a lane may produce: eight per segment of its chunk
    if (cap_lane_out) *cap_lane_out = cap;
    return (size_t)grid * kWarpsPerCta * 32 * cap * sizeof(float2);
}

cudaError_t exact_configure(int kmax) {
    const size_t smem = drop_smem_bytes(kmax);
    cudaError_t e = cudaFuncSetAttribute(k_drop_exact<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_drop_exact<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rows_exact<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rows_exact<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    return e;
}

cudaError_t launch_drop_exact(const DropArgs& a, int grid, cudaStream_t stream) {
    const size_t smem = drop_smem_bytes(a.g.kmax);
    if (a.g.path_model == 1)
        k_drop_exact<true><<<grid, kThreads, smem, stream>>>(a);
    else
        k_drop_exact<false><<<grid, kThreads, smem, stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_rows_exact(const RowsArgs& a, int sms, cudaStream_t stream) {
    const size_t smem = drop_smem_bytes(a.g.kmax);
    long long blocks = (a.count + kWarpsPerCta - 1) / kWarpsPerCta;
    const long long cap = (long long)(sms > 0 ? sms : 148) * 4;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    if (a.g.path_model == 1)
        k_rows_exact<true><<<(int)blocks, kThreads, smem, stream>>>(a);
    else
        k_rows_exact<false><<<(int)blocks, kThreads, smem, stream>>>(a);
    return cudaGetLastError();
}

}  // namespace pct
