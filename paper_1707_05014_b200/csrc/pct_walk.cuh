// pct_walk.cuh -- device functions shared by the kernels of the hot path (pct_kernels.cu: the block engine and the
// inspection kernels): Sigma1^-1 table staging, history loads, the per-warp row
// buffer, the lane-chunked walk of one history by one warp (rule steps 3-4) and the segment-major
// gather (a_i.x) and scatter ((Delta_j, c_j) += ...) passes (R12).
#pragma once
#include <stdio.h>

#include "pct_internal.h"

namespace pct {

// Build with -DPCT_CHECK_BOUNDS for a checking build (compute-sanitizer is closed on this pool: profiles/r2_sanitizers.md):
// every storage slot the walk produces, every row-buffer and table index it forms and every history index it loads
// is tested against its array, violations are counted per kind and reported by bounds_dump().
#ifdef PCT_CHECK_BOUNDS
static __device__ unsigned long long g_pct_bounds[8];  // (one copy per translation unit)
#define PCT_BOUND(kind, ok) do { if (!(ok)) atomicAdd(&g_pct_bounds[kind], 1ULL); else if ((kind) == 0) atomicAdd(&g_pct_bounds[4], 1ULL); } while (0)
// print and clear this translation unit's counters
static inline void bounds_dump_tu(const char* tag) {
    unsigned long long h[8] = {0};
    cudaMemcpyFromSymbol(h, g_pct_bounds, sizeof(h));
    fprintf(stderr, "[bounds %s] segment pairs checked %llu; violations: voxel slot %llu, row buffer %llu, table %llu, history index %llu\n", tag,
            h[4], h[0], h[1], h[2], h[3]);
    for (int i = 0; i < 8; ++i) h[i] = 0;
    cudaMemcpyToSymbol(g_pct_bounds, h, sizeof(h));
}
#else
#define PCT_BOUND(kind, ok)
#endif

#ifndef PCT_WARPS_PER_CTA
#define PCT_WARPS_PER_CTA 10
#endif
#ifndef PCT_CTAS_PER_SM
#define PCT_CTAS_PER_SM 2  // register budget of k_drop_block: 65536 / (2 * 320) -> 102 per thread (95 used)
#endif
#ifndef PCT_BATCH
#define PCT_BATCH 16
#endif
#ifndef PCT_ACC_EVICT_FIRST
#define PCT_ACC_EVICT_FIRST 1  // accumulator traffic of k_update carries an L2 evict_first policy
#endif
#ifndef PCT_WALK_UNROLL
#define PCT_WALK_UNROLL 1
#endif
constexpr int kWalkUnroll = PCT_WALK_UNROLL;  // unroll factor of the walk loop
constexpr int kWarpsPerCta = PCT_WARPS_PER_CTA;
constexpr int kThreads = kWarpsPerCta * 32;
constexpr int kCtasPerSm = PCT_CTAS_PER_SM;
constexpr int kBatch = PCT_BATCH;  // histories a warp takes from the work queue per trip (at most)

// Sigma1^-1 table in shared memory.  Lane l reads the entries of nodes l*C + c: 32 entries C apart per
// 128-bit load, four wavefronts of eight lanes at best.  In a plain layout that best case holds for
// every ODD chunk size C and fails for even ones (C = 8: all lanes in one bank group, 32 wavefronts);
// with entry k at slot k + (k >> 3) it holds for C = 8 (and is fair for the other even sizes) but
// C = 7 degenerates to 24 wavefronts.  No single layout serves both, and C = 7 and C = 8 are two
// thirds of all histories at 256 x 256 x 128, so the table is staged TWICE -- plain and padded -- and a
// history picks its copy by the parity of its C (warp-uniform).  Both copies are padded with zero
// entries up to k = nmin + 33: lanes past the end of a path read (and discard) them.
__host__ __device__ inline int tab_slot(int k) { return k + (k >> 3); }
__host__ __device__ inline int tab_slots(int nmin) { return (tab_slot(nmin + 33) + 4) & ~3; }

__host__ __device__ inline int row_slot(int s);
__host__ __device__ inline int row_slots(int cmax);

// Dynamic shared memory of a CTA: Sigma1^-1 table | PathState[warps][kBatch] | row buffer[warps].
struct SmemLayout {
    int state_off, row_off, row_slots, total;
};
__host__ __device__ inline SmemLayout smem_layout(int nmin) {
    SmemLayout l;
    l.state_off = 4 * (int)sizeof(float4) * tab_slots(nmin);  // two copies of the paired table (two float4 arrays each)
    l.row_off = l.state_off + kWarpsPerCta * kBatch * (int)sizeof(PathState);
    l.row_slots = row_slots((nmin + 32) >> 5);  // K <= nmin: at most ceil((nmin + 1) / 32) segments per lane
    l.total = l.row_off + kWarpsPerCta * l.row_slots * (int)sizeof(float2);
    return l;
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

// Paired layout: the walk evaluates nodes k and k+1 together (mlp_node2), so entry k holds the
// functions of k and of k+1 side by side, ready as 64-bit register pairs:
//   A[k] = (p11[k], p11[k+1], p12[k], p12[k+1]),  B[k] = (p22[k], p22[k+1], s1[k], s1[k+1]).
// s_tab = | A padded | B padded | A plain | B plain |, each of n = tab_slots(nmin) entries.
__device__ __forceinline__ void stage_table(float4* s_tab, const float4* __restrict__ tab, int nmin) {
    const int n = tab_slots(nmin);
    for (int q = threadIdx.x; q < 4 * n; q += kThreads) s_tab[q] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    for (int k = threadIdx.x; k <= nmin; k += kThreads) {
        const float4 a = tab[k];
        const float4 b = k < nmin ? tab[k + 1] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 A = make_float4(a.x, b.x, a.y, b.y), B = make_float4(a.z, b.z, a.w, b.w);
        s_tab[tab_slot(k)] = A;
        s_tab[n + tab_slot(k)] = B;
        s_tab[2 * n + k] = A;
        s_tab[3 * n + k] = B;
    }
    __syncthreads();
}

// Where the inspection kernel wants the row of one history written (all optional).
struct EmitPtrs {
    int32_t* seg_idx;
    float *seg_len, *row_len, *nodes;
};

// ---- row buffer of one warp (shared memory) --------------------------------------------------
// Entry s belongs to segment s of the history being walked: (voxel, length).  voxel = -1: outside
// the grid or past the end of the path (length 0).  The SIGN BIT of the length is the run-head
// flag: set iff the segment starts a run of equal voxels (R10), i.e. iff it counts as one non-zero
// of the row.  The walk writes the buffer lane-chunked (lane l owns segments l*C .. l*C+C-1); the
// gather and scatter passes read it segment-major (lane l takes segments 32 i + l), so that
// neighbouring lanes touch neighbouring voxels and their L2 requests coalesce.  Physical slot
// s + (s >> 5): reads are conflict-free, writes at most 2-way for every chunk size.
__host__ __device__ inline int row_slot(int s) { return s + (s >> 5); }
__host__ __device__ inline int row_slots(int cmax) { return row_slot(32 * cmax) + 2; }

__device__ __forceinline__ void emit_node(const EmitPtrs& em, int k, const float3 a) {
    if (em.nodes) {
        em.nodes[3 * k + 0] = a.x;
        em.nodes[3 * k + 1] = a.y;
        em.nodes[3 * k + 2] = a.z;
    }
}

// Sequential merge of consecutive equal voxels inside one lane (R10) and the lane's part of ||a_i||^2.
struct MergeState {
    int run_idx;      // voxel of the current run (-2: none yet)
    float run_len;    // its length so far (this lane's part)
    float first_len;  // length of the lane's first run (this lane's part), set when the second run starts
    int n_fresh;      // runs started so far (a dropped segment, voxel -1, starts a run here too)
    int nnz;          // run heads with a voxel inside the grid
    float nrm;        // sum of squares of the FINISHED runs
};

// Segment `seg` of the lane (it starts at node `a`), voxel and length known: merge, row-buffer entry.
template <bool EMIT>
__device__ __forceinline__ void take_segment(int lin, float len, const float3 a, int seg, int K, MergeState& m, unsigned row_sa,
                                             const EmitPtrs& em) {
    const bool ok = (seg <= K) && lin >= 0;
    if (EMIT) {  // a dropped segment has no entry in the row; the inspection kernel still reports its length
        if (seg <= K && !ok && em.seg_len) em.seg_len[seg] = len;
    }
    lin = ok ? lin : -1;
    len = ok ? len : 0.0f;
    const bool fresh = lin != m.run_idx;
    if (fresh) {
        m.nrm = __fmaf_rn(m.run_len, m.run_len, m.nrm);  // the finished run
        if (m.n_fresh == 1) m.first_len = m.run_len;
        ++m.n_fresh;
    }
    m.run_len = fresh ? len : m.run_len + len;
    m.run_idx = lin;
    const bool head = fresh && lin >= 0;
    m.nnz += head ? 1 : 0;
    // (an explicit 32-bit shared address: the compiler otherwise rebuilds the buffer's base in every trip)
    asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(row_sa + 8u * (unsigned)row_slot(seg)), "r"(lin),
                 "r"(__float_as_int(head ? -len : len)) : "memory");
    if (EMIT) {
        if (seg <= K) emit_node(em, seg, a);
    }
}

__device__ __forceinline__ float3 lo3(const Node2& n) { return make_float3(lo_of(n.x), lo_of(n.y), lo_of(n.z)); }
__device__ __forceinline__ float3 hi3(const Node2& n) { return make_float3(hi_of(n.x), hi_of(n.y), hi_of(n.z)); }
__device__ __forceinline__ Node2 pair3(const float3 a, const float3 b) {
    Node2 n;
    n.x = pk(a.x, b.x);
    n.y = pk(a.y, b.y);
    n.z = pk(a.z, b.z);
    return n;
}

// Nodes k and k+1 of the path (rule step 3), both halves of one packed evaluation; a node past the
// last interior one is the hull exit point (R9).  k <= 0 gives an unspecified (unused) first half.
template <bool SPLINE>
__device__ __forceinline__ Node2 node_pair(const PathState& st, const float4* s_tab, const float4* s_tabB, int pad_mask, int k,
                                           int K, const float3 exitP) {
    const int slot = k + ((k >> 3) & pad_mask);  // padded copy: tab_slot(k); plain copy: k
    const Node2 n = mlp_node2<SPLINE>(st, s_tab[slot], s_tabB[slot]);
    float3 a = lo3(n), b = hi3(n);
    if (k > K) a = exitP;
    if (k + 1 > K) b = exitP;
    return pair3(a, b);
}

// The two segments a.lo -> b.lo (segment `seg`) and a.hi -> b.hi (segment `seg` + 1): one packed
// evaluation of rule step 4, then the sequential merge.  `first` = false skips the first of them.
template <bool EMIT>
__device__ __forceinline__ void take_two(const Geom& g, const Node2& a, const Node2& b, int seg, bool first, int K, MergeState& m,
                                         unsigned row_sa, const EmitPtrs& em) {
    f2 len, gx, gy, gz;
    segment2(g, a, b, len, gx, gy, gz);
    const int lin_lo = voxel_of(g, lo_of(gx), lo_of(gy), lo_of(gz)), lin_hi = voxel_of(g, hi_of(gx), hi_of(gy), hi_of(gz));
    PCT_BOUND(0, lin_lo >= -1 && lin_lo < g.slice_p * g.nz && lin_hi >= -1 && lin_hi < g.slice_p * g.nz);  // a slot of image / accumulator
    PCT_BOUND(1, (first ? seg : seg + 1) >= 0 && row_slot(seg + 1) < row_slots((g.kmax + 32) >> 5));        // the warp's row buffer
    if (first) take_segment<EMIT>(lin_lo, lo_of(len), lo3(a), seg, K, m, row_sa, em);
    take_segment<EMIT>(lin_hi, hi_of(len), hi3(a), seg + 1, K, m, row_sa, em);
}

// Walk of one history by one warp (steps 3-4 of the rule): fills the warp's row buffer, returns the
// lane's part of ||a_i||^2 and of the non-zero count.
//
// Lane l owns segments k0 .. k0+C-1 (k0 = l*C), i.e. it needs nodes k0 .. k0+C.  Nodes are
// evaluated two at a time (mlp_node2: packed fp32, one instruction for both).  The lane evaluates
// its LAST two nodes (k0+C-1, k0+C) first and hands the last one to lane l+1 as that lane's start
// node with one shuffle (lane 0 starts at the hull entry point), then walks the node pairs
// (k0+1, k0+2), (k0+3, k0+4), ... -- two segments per trip -- up to node k0+C-2, and finishes with
// the one or two segments that end at the nodes it evaluated first.  The MLP node at depth k*h is
// closed-form in k, there is no recurrence along the path.  Lanes past the end of the path run the
// same instructions on harmless values and are masked.
template <bool EMIT, bool SPLINE>
__device__ __forceinline__ void walk_history(const Geom& g, const PathState& S, const float4* s_tab, int lane, float2* row,
                                             float& nrm, int& nnz, const EmitPtrs& em) {
    const PathState st = S;  // shared memory -> registers, once per history
    const int K = st.K;
    const int C = (K + 32) >> 5;  // ceil((K + 1) / 32) segments per lane
    const int tab_n = tab_slots(g.kmax);
    const int pad_mask = (C & 1) ? 0 : -1;  // odd C: the plain copy of the table, even C: the padded one
    const float4* s_tabA = s_tab + ((C & 1) ? 2 * tab_n : 0);
    const float4* s_tabB = s_tabA + tab_n;
    const int k0 = lane * C;
    PCT_BOUND(2, tab_slot(k0 + C - 1) < tab_n && C <= ((g.kmax + 32) >> 5));  // the staged table (its last entry read by this lane)
    const float3 exitP = to_object(st, st.t2, st.u2, st.v2);  // node K+1: the hull exit point, assigned (R9)
    const Node2 Z = node_pair<SPLINE>(st, s_tabA, s_tabB, pad_mask, k0 + C - 1, K, exitP);
    const float3 last = hi3(Z);
    float3 prv;
    prv.x = __shfl_up_sync(0xffffffffu, last.x, 1);
    prv.y = __shfl_up_sync(0xffffffffu, last.y, 1);
    prv.z = __shfl_up_sync(0xffffffffu, last.z, 1);
    if (lane == 0) prv = to_object(st, st.t0, st.u0, st.v0);  // node 0: the hull entry point (R9)
    MergeState m{-2, 0.0f, 0.0f, 0, 0, 0.0f};
    const unsigned row_sa = (unsigned)__cvta_generic_to_shared(row);
    int c = 1;  // next node of the lane to evaluate; segments k0 .. k0+c-2 are done
#pragma unroll kWalkUnroll
    for (; c <= C - 2; c += 2) {
        const Node2 N = node_pair<SPLINE>(st, s_tabA, s_tabB, pad_mask, k0 + c, K, exitP);
        take_two<EMIT>(g, pair3(prv, lo3(N)), N, k0 + c - 1, true, K, m, row_sa, em);
        prv = hi3(N);
    }
    {  // the last two segments (C - c + 1 == 2: via node k0+C-1) or the last one (prv IS node k0+C-1)
        const bool two = C - c + 1 == 2;
        const float3 mid = two ? lo3(Z) : prv;
        take_two<EMIT>(g, pair3(prv, mid), pair3(mid, last), k0 + C - 2, two, K, m, row_sa, em);
    }
    if (EMIT) {
        if (k0 <= K && K < k0 + C) emit_node(em, K + 1, exitP);
    }
    m.nrm = __fmaf_rn(m.run_len, m.run_len, m.nrm);
    const bool whole = m.n_fresh == 1;  // the lane's whole chunk is one run
    if (whole) m.first_len = m.run_len;
    // ---- lane seams: the lane's first run may continue the previous lane's last run ----------
    // With p = this lane's part and q = the part in earlier lanes, (q + p)^2 = q^2 + 2qp + p^2:
    // q^2 is already in the earlier lanes' sums, p^2 in this lane's, the seam adds 2qp.
    const float2 e0 = row[row_slot(k0)];
    const int lin0 = __float_as_int(e0.x);
    const int prev_idx = __shfl_up_sync(0xffffffffu, m.run_idx, 1);
    const float prev_len = __shfl_up_sync(0xffffffffu, m.run_len, 1);
    const bool prev_whole = __shfl_up_sync(0xffffffffu, (int)whole, 1) != 0;
    const bool cont = lane > 0 && lin0 >= 0 && lin0 == prev_idx;
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
        row[row_slot(k0)] = make_float2(e0.x, fabsf(e0.y));  // not a run head after all
        --m.nnz;
        m.nrm = __fmaf_rn(2.0f * carry, m.first_len, m.nrm);
    }
    nrm = m.nrm;
    nnz = m.nnz;
    __syncwarp();  // the row buffer is complete: the passes below read it segment-major
}

// ---- segment-major passes over the row buffer ------------------------------------------------
// Lane l reads segments 32 i + l: physical slot row_slot(32 i + l) = 33 i + l.  The passes are
// instantiated for an exact number N of segments per lane (no per-slot bounds test) and
// dispatched on the warp-uniform C.

// (Delta_j, c_j) += (v, cnt): one 64-bit vector reduction, no return value, predicated on lin >= 0.
__device__ __forceinline__ void red_add_v2(float2* acc, int lin, float v, float cnt) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .u64 ad;\n\t"
        "setp.ge.s32 p, %1, 0;\n\t"
        "mad.wide.s32 ad, %1, 8, %0;\n\t"
        "@p red.global.add.v2.f32 [ad], {%2, %3};\n\t}"
        :: "l"(acc), "r"(lin), "f"(v), "f"(cnt) : "memory");
}

// L2 residency.  The image (4 B/voxel) and the accumulator (8 B/voxel) together do not stay in the
// L2 across the two kernels of a DROP block (100 MB at 256 x 256 x 128 against 126 MB split over two
// dies), so both kernels kept re-reading them from HBM and one gather in three paid the DRAM latency.
// Every access to the IMAGE carries an evict_last policy, the accumulator traffic stays evict_normal:
// the image stays resident, the gather always hits the L2.
__device__ __forceinline__ unsigned long long policy_evict_last() {
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ unsigned long long policy_evict_first() {
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ float ld_image(const float* p, unsigned long long pol) {
    float v;
    asm volatile("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}

template <int N>
__device__ __forceinline__ float gather_n(const float2* rl, const float* __restrict__ x) {
    float2 e[N];
    float xv[N];
    const unsigned long long pol = policy_evict_last();
#pragma unroll
    for (int u = 0; u < N; ++u) e[u] = rl[33 * u];
#pragma unroll
    for (int u = 0; u < N; ++u) {
        const int lin = __float_as_int(e[u].x);
        xv[u] = 0.0f;
        if (lin >= 0) xv[u] = ld_image(x + lin, pol);
    }
    float dot = 0.0f;
#pragma unroll
    for (int u = 0; u < N; ++u) dot = __fmaf_rn(fabsf(e[u].y), xv[u], dot);
    return dot;
}

template <int N>
__device__ __forceinline__ void scatter_n(const float2* rl, float2* acc, float r) {
#pragma unroll
    for (int u = 0; u < N; ++u) {
        const float2 e = rl[33 * u];
        red_add_v2(acc, __float_as_int(e.x), r * fabsf(e.y), __float_as_int(e.y) < 0 ? 1.0f : 0.0f);
    }
}

#define PCT_SWITCH_N(n, CALL)        \
    switch (n) {                     \
        case 1: CALL(1); break;      \
        case 2: CALL(2); break;      \
        case 3: CALL(3); break;      \
        case 4: CALL(4); break;      \
        case 5: CALL(5); break;      \
        case 6: CALL(6); break;      \
        case 7: CALL(7); break;      \
        default: break;              \
    }

// a_i.x (a4): gather of x through L2, C segments per lane.
__device__ __forceinline__ float gather_row(const float2* row, int lane, int C, const float* __restrict__ x) {
    const float2* rl = row + lane;
    float dot = 0.0f;
    int i = 0;
    for (; i + 8 <= C; i += 8) dot += gather_n<8>(rl + 33 * i, x);
#define PCT_G(N) dot += gather_n<N>(rl + 33 * i, x)
    PCT_SWITCH_N(C - i, PCT_G);
#undef PCT_G
    return dot;
}

// scatter (a5): (Delta_j, c_j) += (r a_ij, 1 per run head).
__device__ __forceinline__ void scatter_row(const float2* row, int lane, int C, float2* acc, float r) {
    const float2* rl = row + lane;
    int i = 0;
    for (; i + 8 <= C; i += 8) scatter_n<8>(rl + 33 * i, acc, r);
#define PCT_S(N) scatter_n<N>(rl + 33 * i, acc, r)
    PCT_SWITCH_N(C - i, PCT_S);
#undef PCT_S
}

}  // namespace pct
