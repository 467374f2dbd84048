// pct_walk16.cuh -- the walk, gather and scatter of pct_walk.cuh for TWO histories per warp, sixteen lanes each.
//
// One warp per history spends 28 % of its instructions on work that does not grow with the path (state load, lane seams,
// the two warp sums, the residual, pass set-up: profiles/r2a_ncu_full.md) and rounds every path up to a multiple of 64
// segments (32 lanes x a node pair).  Here a warp walks two histories side by side: lanes 0-15 one, lanes 16-31 the other,
// with ONE chunk size C = ceil((max(K_a, K_b) + 1) / 16) for both (so loops, table copy and pass sizes stay
// warp-uniform; the shorter path's lanes past its end produce empty entries), every shuffle 16 lanes wide.  The
// per-history fixed work is issued once for two histories and a path is rounded up to a multiple of 32 segments.
// The arithmetic of a segment is the same device code (node_pair, take_two): the rows are the same rows.
#pragma once
#include "pct_walk.cuh"

namespace pct {

__device__ __forceinline__ float half_sum(float v) {  // sum over the 16 lanes of a half warp
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, 16);
    return v;
}

// Row buffer of one history in this mapping: segment s at slot s + (s >> 5) as before; most segments per lane:
// ceil((kmax + 1) / 16).
__host__ __device__ inline int row16_slots(int kmax) { return row_slot(16 * ((kmax + 16) >> 4)) + 2; }

// Walk of the history `S` by the 16 lanes of one half warp (hl = lane & 15) with chunk size C >= ceil((K + 1) / 16):
// walk_history of pct_walk.cuh with 16-lane shuffles.  Both halves of the warp call it together with the same C.
template <bool SPLINE>
__device__ __forceinline__ void walk_history16(const Geom& g, const PathState& S, const float4* s_tab, int hl, int C, float2* row,
                                               float& nrm, int& nnz) {
    const PathState st = S;
    const int K = st.K;
    const int tab_n = tab_slots(g.kmax);
    const int pad_mask = (C & 1) ? 0 : -1;
    const float4* s_tabA = s_tab + ((C & 1) ? 2 * tab_n : 0);
    const float4* s_tabB = s_tabA + tab_n;
    const int k0 = hl * C;
    PCT_BOUND(2, tab_slot(k0 + C - 1) < tab_n && C <= ((g.kmax + 16) >> 4));
    const float3 exitP = to_object(st, st.t2, st.u2, st.v2);
    const Node2 Z = node_pair<SPLINE>(st, s_tabA, s_tabB, pad_mask, k0 + C - 1, K, exitP);
    const float3 last = hi3(Z);
    float3 prv;
    prv.x = __shfl_up_sync(0xffffffffu, last.x, 1, 16);
    prv.y = __shfl_up_sync(0xffffffffu, last.y, 1, 16);
    prv.z = __shfl_up_sync(0xffffffffu, last.z, 1, 16);
    if (hl == 0) prv = to_object(st, st.t0, st.u0, st.v0);
    MergeState m{-2, 0.0f, 0.0f, 0, 0, 0.0f};
    const unsigned row_sa = (unsigned)__cvta_generic_to_shared(row);
    const EmitPtrs no_emit{nullptr, nullptr, nullptr, nullptr};
    int c = 1;
#pragma unroll kWalkUnroll
    for (; c <= C - 2; c += 2) {
        const Node2 N = node_pair<SPLINE>(st, s_tabA, s_tabB, pad_mask, k0 + c, K, exitP);
        take_two<false>(g, pair3(prv, lo3(N)), N, k0 + c - 1, true, K, m, row_sa, no_emit);
        prv = hi3(N);
    }
    {
        const bool two = C - c + 1 == 2;
        const float3 mid = two ? lo3(Z) : prv;
        take_two<false>(g, pair3(prv, mid), pair3(mid, last), k0 + C - 2, two, K, m, row_sa, no_emit);
    }
    m.nrm = __fmaf_rn(m.run_len, m.run_len, m.nrm);
    const bool whole = m.n_fresh == 1;
    if (whole) m.first_len = m.run_len;
    // lane seams, inside the half warp
    const float2 e0 = row[row_slot(k0)];
    const int lin0 = __float_as_int(e0.x);
    const int prev_idx = __shfl_up_sync(0xffffffffu, m.run_idx, 1, 16);
    const float prev_len = __shfl_up_sync(0xffffffffu, m.run_len, 1, 16);
    const bool prev_whole = __shfl_up_sync(0xffffffffu, (int)whole, 1, 16) != 0;
    const bool cont = hl > 0 && lin0 >= 0 && lin0 == prev_idx;
    const float base = cont ? prev_len : 0.0f;
    float carry = base;
    if (__any_sync(0xffffffffu, cont && prev_whole)) {
        for (int it = 0; it < 15; ++it) {
            const float up = __shfl_up_sync(0xffffffffu, carry, 1, 16);
            const float nc = (cont && prev_whole) ? base + up : base;
            const bool changed = nc != carry;
            carry = nc;
            if (!__any_sync(0xffffffffu, changed)) break;
        }
    }
    if (cont) {
        row[row_slot(k0)] = make_float2(e0.x, fabsf(e0.y));
        --m.nnz;
        m.nrm = __fmaf_rn(2.0f * carry, m.first_len, m.nrm);
    }
    nrm = m.nrm;
    nnz = m.nnz;
    __syncwarp();
}

// Segment-major passes: lane hl reads segments 16 u + hl of its history, slot 16 u + (u >> 1) + hl.  N consecutive
// rounds from an EVEN round u0 (rl already points at its slot): offsets 16 v + (v >> 1).
template <int N>
__device__ __forceinline__ float gather16_n(const float2* rl, const float* __restrict__ x) {
    float2 e[N];
    float xv[N];
    const unsigned long long pol = policy_evict_last();
#pragma unroll
    for (int v = 0; v < N; ++v) e[v] = rl[16 * v + (v >> 1)];
#pragma unroll
    for (int v = 0; v < N; ++v) {
        const int lin = __float_as_int(e[v].x);
        xv[v] = 0.0f;
        if (lin >= 0) xv[v] = ld_image(x + lin, pol);
    }
    float dot = 0.0f;
#pragma unroll
    for (int v = 0; v < N; ++v) dot = __fmaf_rn(fabsf(e[v].y), xv[v], dot);
    return dot;
}

template <int N>
__device__ __forceinline__ void scatter16_n(const float2* rl, float2* acc, float r, bool on) {
#pragma unroll
    for (int v = 0; v < N; ++v) {
        const float2 e = rl[16 * v + (v >> 1)];
        red_add_v2(acc, on ? __float_as_int(e.x) : -1, r * fabsf(e.y), __float_as_int(e.y) < 0 ? 1.0f : 0.0f);
    }
}

// a_i.x of the half's history: C rounds (C is the warp's common chunk size = rounds per lane).
__device__ __forceinline__ float gather16_row(const float2* row, int hl, int C, const float* __restrict__ x) {
    const float2* rl = row + hl;
    float dot = 0.0f;
    int i = 0;
    for (; i + 8 <= C; i += 8) dot += gather16_n<8>(rl + 132 * (i >> 3), x);  // (eight rounds are 128 segments + 4 pad slots)
#define PCT_G16(N) dot += gather16_n<N>(rl + 132 * (i >> 3), x)
    PCT_SWITCH_N(C - i, PCT_G16);
#undef PCT_G16
    return dot;
}

__device__ __forceinline__ void scatter16_row(const float2* row, int hl, int C, float2* acc, float r, bool on) {
    const float2* rl = row + hl;
    int i = 0;
    for (; i + 8 <= C; i += 8) scatter16_n<8>(rl + 132 * (i >> 3), acc, r, on);
#define PCT_S16(N) scatter16_n<N>(rl + 132 * (i >> 3), acc, r, on)
    PCT_SWITCH_N(C - i, PCT_S16);
#undef PCT_S16
}

// Sort of up to 16 keys held by lanes 0-15 (one each), ascending; both halves of the warp sort their own copy.  Bitonic
// network, ten compare-exchange steps.
__device__ __forceinline__ int sort16(int key, int hl) {
#pragma unroll
    for (int k = 2; k <= 16; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
            const int other = __shfl_xor_sync(0xffffffffu, key, j, 16);
            const bool up = (hl & k) == 0;       // direction of this lane's block
            const bool lower = (hl & j) == 0;    // this lane keeps the smaller of the two when ascending
            const int mn = key < other ? key : other, mx = key < other ? other : key;
            key = (lower == up) ? mn : mx;
        }
    }
    return key;
}

}  // namespace pct
