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
#include "pct_internal.h"

namespace pct {

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

size_t drop_smem_bytes(int nmin) { return (size_t)smem_layout(nmin).total; }

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
    if (first) take_segment<EMIT>(voxel_of(g, lo_of(gx), lo_of(gy), lo_of(gz)), lo_of(len), lo3(a), seg, K, m, row_sa, em);
    take_segment<EMIT>(voxel_of(g, hi_of(gx), hi_of(gy), hi_of(gz)), hi_of(len), hi3(a), seg + 1, K, m, row_sa, em);
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
    const int tab_n = tab_slots(g.nmin);
    const int pad_mask = (C & 1) ? 0 : -1;  // odd C: the plain copy of the table, even C: the padded one
    const float4* s_tabA = s_tab + ((C & 1) ? 2 * tab_n : 0);
    const float4* s_tabB = s_tabA + tab_n;
    const int k0 = lane * C;
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
constexpr int kPhases = 4;
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
    const SmemLayout lay = smem_layout(g.nmin);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * lay.row_slots;
    __shared__ Queue q;  // one copy per CTA: the phase of a ticket is looked up by index
    if (threadIdx.x == 0) {
        long long first = a.first, count = a.count;
        if (first < 0) {
            first = a.ctrl->block * a.block_size;
            count = a.n - first < a.block_size ? a.n - first : a.block_size;
        }
        q = make_queue(first, count, (long long)gridDim.x * kWarpsPerCta);
        q.interleave = a.first < 0 && a.order != nullptr;
    }
    stage_table(s_tab, a.tab, g.nmin);  // (ends with __syncthreads: q is visible)
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

cudaError_t drop_configure(int nmin, int* grid_out) {
    if (((nmin + 32) >> 5) > 64) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(nmin);
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_drop_block<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_drop_block<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_drop_block<false>, kThreads, smem);
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
    if (a.g.path_model == 1)
        k_drop_block<true><<<grid, kThreads, smem, stream>>>(a);
    else
        k_drop_block<false><<<grid, kThreads, smem, stream>>>(a);
    return cudaGetLastError();
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
__global__ void __launch_bounds__(256) k_update(float* __restrict__ x, float2* __restrict__ acc, long long n_voxels,
                                                float lambda, Ctrl* ctrl, long long n_blocks) {
    constexpr int UN = PCT_UPD_UNROLL;
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
            const long long q = q0 + u * stride;
            if (q < n4) {
                a01[u] = PCT_LD_ACC(a4 + 2 * q);
                a23[u] = PCT_LD_ACC(a4 + 2 * q + 1);
                xv[u] = ld4_hint(x4 + q, keep);
            } else {
                a01[u] = a23[u] = xv[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const long long q = q0 + u * stride;
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
                          cudaStream_t stream) {
    const long long n4 = n_voxels >> 2;
    long long blocks = (n4 + 256 * PCT_UPD_UNROLL - 1) / (256 * PCT_UPD_UNROLL);
    if (blocks < 1) blocks = 1;
    if (blocks > 148 * PCT_UPD_CTAS) blocks = 148 * PCT_UPD_CTAS;
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
template <bool SPLINE>
__global__ void __launch_bounds__(kThreads) k_rows(const RowsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const SmemLayout lay = smem_layout(g.nmin);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * lay.row_slots;
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
            float nrm;
            int nnz;
            walk_history<true, SPLINE>(g, S, s_tab, lane, row, nrm, nnz, em);
            nnz_total = __reduce_add_sync(0xffffffffu, nnz);
            // the row as the hot path sees it: read back from the row buffer, segment-major
            for (int k = lane; k <= K; k += 32) {
                const float2 e = row[row_slot(k)];
                if (em.seg_idx) em.seg_idx[k] = __float_as_int(e.x);
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

cudaError_t launch_rows(const RowsArgs& a, cudaStream_t stream) {
    if (((a.g.nmin + 32) >> 5) > 64) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(a.g.nmin);
    long long blocks = (a.count + kWarpsPerCta - 1) / kWarpsPerCta;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    cudaError_t e = cudaSuccess;
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
    const long long grid = n_blocks < 148 * 4 ? n_blocks : 148 * 4;
    k_order_blocks<<<(int)grid, 512, 0, stream>>>(H, g, n, block_size, first_block, n_blocks, n_slabs, order);
    return cudaGetLastError();
}

// CARP (R29): the new solution is the arithmetic mean of the P string solutions, voxel by
// voxel; summed in the order of the strings (deterministic).  xs = P images of n voxels, back to back.
__global__ void __launch_bounds__(256) k_mean(float* __restrict__ x, const float* __restrict__ xs, int n_strings, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    const float fp = (float)n_strings;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        float s = 0.0f;
        for (int p = 0; p < n_strings; ++p) s += xs[(long long)p * n + j];
        x[j] = __fdiv_rn(s, fp);
    }
}

cudaError_t launch_mean(float* x, const float* xs, int n_strings, long long n, cudaStream_t stream) {
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    k_mean<<<(int)blocks, 256, 0, stream>>>(x, xs, n_strings, n);
    return cudaGetLastError();
}

}  // namespace pct
