// pct_tvs.cu -- total-variation superiorization step on the image ("both
// algorithms incorporate total variation superiorization (TVS), which 'jiggles' the solution ... In CARP, TVS is applied
// just once to the initial solution at the start of each iteration.  In DROP, however, TVS is applied to the initial
// solution that enters each block").  The paper prints no formula; R31 fixes the step:
//
//   TV(x) = sum_ijk sqrt(dx^2 + dy^2 + dz^2 + eps^2)  (forward differences, zero across the far faces, eps = 1e-6)
//   g = grad TV(x);  v = -g / ||g||;  z_l = x + beta 2^-l v, l = 0 .. n_half-1;  x <- the first z_l with TV(z_l) <= TV(x)
//   beta <- gamma * (the step that was taken, or beta 2^-n_half if none was)
//
// Three launches per step, all on the image in its storage order (voxel_slot: 2 x 2 in-plane tiles):
//   k_tv_grad   g and the fp64 sums TV(x), ||g||^2;
//   k_tv_probe  TV(z_l) for every level at once (z is never stored: its differences follow from those of x and g);
//   k_tv_apply  picks the level from the sums (every thread, identically), moves the image, zeroes the other step's sums.
// A thread of the two stencil kernels owns one 2 x 2 tile (ONE 16 B load per slice) and marches along z over a chunk of
// slices, a warp 32 tiles of a tile row: the x neighbours come from the next lane, the y neighbours from one 8 B load of
// the next tile row, the z neighbours from the slice already in registers; one reciprocal square root per term.  (A
// thread per voxel computing voxel_slot for each of its 13 neighbours issued 233 warp instructions per 32 voxels and ran
// at the issue limit: profiles/r2f_tvs.md.)
// Terms are formed in fp32, summed in fp64 (per thread, block tree, then one atomic per block): the comparison
// TV(z) <= TV(x) is taken on sums whose rounding is far below the change a step makes.
#include <algorithm>

#include "pct_internal.h"

namespace pct {

constexpr float kTvEps2 = 1.0e-12f;  // eps^2
constexpr int kTvThreads = 256;

__device__ __forceinline__ float rsq(float q) {  // q >= eps^2 > 0: no special cases (relative error 2^-22)
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(q));
    return r;
}

// One term of TV: voxel value c, its +x, +y, +z neighbours (a neighbour outside the grid is passed as c: difference 0).
// r d / t are the partial derivatives of the term t with respect to the three neighbours.
struct Term {
    float rdx, rdy, rdz, t;
};
__device__ __forceinline__ Term term(float c, float xr, float xu, float xz) {
    const float dx = xr - c, dy = xu - c, dz = xz - c;
    const float q = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, kTvEps2)));
    const float r = rsq(q);
    Term o;
    o.rdx = dx * r;
    o.rdy = dy * r;
    o.rdz = dz * r;
    o.t = q * r;
    return o;
}

__device__ __forceinline__ double block_sum(double v, double* s_part) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();  // (s_part may still be read from the previous call)
    if (lane == 0) s_part[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (warp == 0) {
        t = lane < (int)(blockDim.x >> 5) ? s_part[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;  // valid in thread 0
}

// Work items of the stencil kernels: (chunk of slices, tile row, group of 32 tiles), one warp each.
struct TvItems {
    int nxt, nyt;       // tiles per tile row, tile rows per slice
    int wx_n;           // warps per tile row
    int chunk, n_items;
};

// What a lane needs to know about its tile, the same for every slice.
struct TileLane {
    bool t_ok;                // the tile exists (lanes past the end of the tile row work on a copy of the last tile)
    bool vi1, vi2, vj1, vj2;  // voxels i + 1, i + 2 (i = 2 it), j + 1, j + 2 (j = 2 jt) are inside the grid
    int it, jt, k0, k1;
    long long own, right;     // slot of the tile and of its right neighbour within a slice
};
__device__ __forceinline__ TileLane tile_lane(const Geom& g, const TvItems& w, int item, int lane) {
    TileLane a;
    const int per_chunk = w.wx_n * w.nyt;
    const int kc = item / per_chunk, rem = item - kc * per_chunk;
    a.jt = rem / w.wx_n;
    a.it = 32 * (rem - a.jt * w.wx_n) + lane;
    a.t_ok = a.it < w.nxt;
    const int itc = a.t_ok ? a.it : w.nxt - 1;
    a.vi1 = 2 * itc + 1 < g.nx;
    a.vi2 = 2 * itc + 2 < g.nx;
    a.vj1 = 2 * a.jt + 1 < g.ny;
    a.vj2 = 2 * a.jt + 2 < g.ny;
    a.k0 = kc * w.chunk;
    a.k1 = a.k0 + w.chunk < g.nz ? a.k0 + w.chunk : g.nz;
    a.own = (long long)a.jt * 2 * g.nxp + 4 * itc;
    a.right = a.own + (itc + 1 < w.nxt ? 4 : 0);
    return a;
}

__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float2 ld2(const float* p) { return __ldg(reinterpret_cast<const float2*>(p)); }

// Entries 0 and 2 of the right neighbour tile: the next lane's, the last lane loads them.
__device__ __forceinline__ void right_column(const float4& P, const float* slice, const TileLane& a, int lane, float& r0, float& r2) {
    r0 = __shfl_down_sync(0xffffffffu, P.x, 1);
    r2 = __shfl_down_sync(0xffffffffu, P.z, 1);
    if (lane == 31) {
        const float4 R = ld4(slice + a.right);
        r0 = R.x;
        r2 = R.z;
    }
}

__global__ void __launch_bounds__(kTvThreads) k_tv_grad(const float* __restrict__ x, float* __restrict__ grad, const Geom g,
                                                        const TvItems w, TvState* st, int parity) {
    __shared__ double s_part[kTvThreads / 32];
    double tv = 0.0, g2 = 0.0;
    const int lane = threadIdx.x & 31;
    const int warps = (gridDim.x * kTvThreads) >> 5;
    const long long up_row = 2LL * g.nxp;
    for (int item = (blockIdx.x * kTvThreads + threadIdx.x) >> 5; item < w.n_items; item += warps) {
        const TileLane a = tile_lane(g, w, item, lane);
        const bool has_d = a.jt > 0;
        const int ks = a.k0 > 0 ? a.k0 - 1 : 0;  // one slice below the chunk: its d/dz terms enter the chunk's first slice
        const float* sl = x + (long long)ks * g.slice_p;
        float4 P = ld4(sl + a.own);
        float2 D = has_d ? ld2(sl + a.own - up_row + 2) : make_float2(0.f, 0.f);  // entries 2, 3 of the tile below in y
        float z0 = 0.f, z1 = 0.f, z2 = 0.f, z3 = 0.f;                             // r dz of the slice below
        for (int k = ks; k < a.k1; ++k, sl += g.slice_p) {
            const bool top = k + 1 >= g.nz;
            const float4 Pn = top ? P : ld4(sl + g.slice_p + a.own);
            const float2 U = a.vj2 ? ld2(sl + a.own + up_row) : make_float2(0.f, 0.f);  // entries 0, 1 of the tile above in y
            float r0, r2;
            right_column(P, sl, a, lane, r0, r2);
            const Term T0 = term(P.x, a.vi1 ? P.y : P.x, a.vj1 ? P.z : P.x, Pn.x);
            const Term T1 = term(P.y, a.vi2 ? r0 : P.y, a.vj1 ? P.w : P.y, Pn.y);
            const Term T2 = term(P.z, a.vi1 ? P.w : P.z, a.vj2 ? U.x : P.z, Pn.z);
            const Term T3 = term(P.w, a.vi2 ? r2 : P.w, a.vj2 ? U.y : P.w, Pn.w);
            float2 Dn = D;
            if (has_d && !top) Dn = ld2(sl + g.slice_p + a.own - up_row + 2);
            if (k >= a.k0) {
                // d t(i-1) / d x(i): voxels 1, 3 of the left tile, the previous lane's terms; lane 0 forms them itself
                float lx1 = __shfl_up_sync(0xffffffffu, T1.rdx, 1), lx3 = __shfl_up_sync(0xffffffffu, T3.rdx, 1);
                if (lane == 0) {
                    lx1 = lx3 = 0.f;
                    if (a.it > 0) {
                        const float4 L = ld4(sl + a.own - 4);
                        const float4 Ln = top ? L : ld4(sl + g.slice_p + a.own - 4);
                        const float ulc = a.vj2 ? __ldg(sl + a.own - 4 + up_row + 1) : 0.f;
                        lx1 = term(L.y, P.x, a.vj1 ? L.w : L.y, Ln.y).rdx;
                        lx3 = term(L.w, P.z, a.vj2 ? ulc : L.w, Ln.w).rdx;
                    }
                }
                // d t(j-1) / d x(j): voxels 2, 3 of the tile below in y, formed here
                float dy2 = 0.f, dy3 = 0.f;
                if (has_d) {
                    float dr2 = __shfl_down_sync(0xffffffffu, D.x, 1);
                    if (lane == 31) dr2 = __ldg(sl + a.right - up_row + 2);
                    dy2 = term(D.x, a.vi1 ? D.y : D.x, P.x, Dn.x).rdy;
                    dy3 = term(D.y, a.vi2 ? dr2 : D.y, P.y, Dn.y).rdy;
                }
                const bool ok1 = a.vi1, ok2 = a.vj1, ok3 = a.vi1 && a.vj1;
                float4 gv;
                gv.x = lx1 + dy2 + z0 - (T0.rdx + T0.rdy + T0.rdz);
                gv.y = ok1 ? T0.rdx + dy3 + z1 - (T1.rdx + T1.rdy + T1.rdz) : 0.f;
                gv.z = ok2 ? lx3 + T0.rdy + z2 - (T2.rdx + T2.rdy + T2.rdz) : 0.f;
                gv.w = ok3 ? T2.rdx + T1.rdy + z3 - (T3.rdx + T3.rdy + T3.rdz) : 0.f;
                if (a.t_ok) {
                    *reinterpret_cast<float4*>(grad + (sl - x) + a.own) = gv;
                    tv += (double)(T0.t + (ok1 ? T1.t : 0.f) + (ok2 ? T2.t : 0.f) + (ok3 ? T3.t : 0.f));
                    g2 += (double)fmaf(gv.x, gv.x, fmaf(gv.y, gv.y, fmaf(gv.z, gv.z, gv.w * gv.w)));
                }
            }
            z0 = T0.rdz, z1 = T1.rdz, z2 = T2.rdz, z3 = T3.rdz;
            P = Pn;
            D = Dn;
        }
    }
    const double sa = block_sum(tv, s_part);
    const double sb = block_sum(g2, s_part);
    if (threadIdx.x == 0) {
        atomicAdd(&st->sums[parity].tvx, sa);
        atomicAdd(&st->sums[parity].g2, sb);
    }
}

__device__ __forceinline__ float keep_if(bool on, float v) {  // on ? v : 0 as one select (never a branch around the arithmetic)
    float r;
    asm("{ .reg .pred p; setp.ne.s32 p, %2, 0; selp.f32 %0, %1, 0f00000000, p; }" : "=f"(r) : "f"(v), "r"((int)on));
    return r;
}

// One voxel of the probe: forward differences a of x and b of g; adds |a - s 2^-l b| for NH levels, s the first one's,
// to acc.
template <int NH>
__device__ __forceinline__ void probe_voxel(float c, float xr, float xu, float xz, float gc, float gr, float gu, float gz, float s0,
                                            bool on, float (&acc)[NH]) {
    const float ax = xr - c, ay = xu - c, az = xz - c;
    const float bx = gr - gc, by = gu - gc, bz = gz - gc;
    float sl = s0;
#pragma unroll
    for (int l = 0; l < NH; ++l) {
        const float dx = fmaf(-sl, bx, ax), dy = fmaf(-sl, by, ay), dz = fmaf(-sl, bz, az);
        const float q = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, kTvEps2)));
        acc[l] += keep_if(on, q * rsq(q));
        sl *= 0.5f;
    }
}

// TV(z_l) for the NH levels from l0 on.  The step takes the FIRST level that does not raise the total variation, and that
// is nearly always level 0: level 0 is probed by a launch of its own, and the launch for the other levels returns at once
// when an earlier level already qualifies (its sums are then never read).
template <int NH>
__global__ void __launch_bounds__(kTvThreads) k_tv_probe(const float* __restrict__ x, const float* __restrict__ grad, const Geom g,
                                                         const TvItems w, TvState* st, int parity, int l0) {
    __shared__ double s_part[kTvThreads / 32];
    const double g2 = st->sums[parity].g2;
    if (!(g2 > 0.0)) return;  // flat image: no direction, no step
    for (int l = 0; l < l0; ++l)
        if (st->sums[parity].tvz[l] <= st->sums[parity].tvx) return;
    float s0 = st->beta[parity] / (float)sqrt(g2);  // z = x - s g,  s = beta 2^-l / ||g||
    for (int l = 0; l < l0; ++l) s0 *= 0.5f;
    double tz[NH];
#pragma unroll
    for (int l = 0; l < NH; ++l) tz[l] = 0.0;
    const int lane = threadIdx.x & 31;
    const int warps = (gridDim.x * kTvThreads) >> 5;
    const long long up_row = 2LL * g.nxp;
    for (int item = (blockIdx.x * kTvThreads + threadIdx.x) >> 5; item < w.n_items; item += warps) {
        const TileLane a = tile_lane(g, w, item, lane);
        const bool ok1 = a.t_ok && a.vi1, ok2 = a.t_ok && a.vj1, ok3 = ok1 && a.vj1;
        const float* sx = x + (long long)a.k0 * g.slice_p;
        const float* sg = grad + (long long)a.k0 * g.slice_p;
        float4 P = ld4(sx + a.own), G = ld4(sg + a.own);
        for (int k = a.k0; k < a.k1; ++k, sx += g.slice_p, sg += g.slice_p) {
            const bool top = k + 1 >= g.nz;
            const float4 Pn = top ? P : ld4(sx + g.slice_p + a.own);
            const float4 Gn = top ? G : ld4(sg + g.slice_p + a.own);
            const float2 U = a.vj2 ? ld2(sx + a.own + up_row) : make_float2(0.f, 0.f);
            const float2 V = a.vj2 ? ld2(sg + a.own + up_row) : make_float2(0.f, 0.f);
            float r0, r2, q0, q2;
            right_column(P, sx, a, lane, r0, r2);
            right_column(G, sg, a, lane, q0, q2);
            float acc[NH];
#pragma unroll
            for (int l = 0; l < NH; ++l) acc[l] = 0.f;
            probe_voxel<NH>(P.x, a.vi1 ? P.y : P.x, a.vj1 ? P.z : P.x, Pn.x, G.x, a.vi1 ? G.y : G.x, a.vj1 ? G.z : G.x, Gn.x, s0, a.t_ok, acc);
            probe_voxel<NH>(P.y, a.vi2 ? r0 : P.y, a.vj1 ? P.w : P.y, Pn.y, G.y, a.vi2 ? q0 : G.y, a.vj1 ? G.w : G.y, Gn.y, s0, ok1, acc);
            probe_voxel<NH>(P.z, a.vi1 ? P.w : P.z, a.vj2 ? U.x : P.z, Pn.z, G.z, a.vi1 ? G.w : G.z, a.vj2 ? V.x : G.z, Gn.z, s0, ok2, acc);
            probe_voxel<NH>(P.w, a.vi2 ? r2 : P.w, a.vj2 ? U.y : P.w, Pn.w, G.w, a.vi2 ? q2 : G.w, a.vj2 ? V.y : G.w, Gn.w, s0, ok3, acc);
#pragma unroll
            for (int l = 0; l < NH; ++l) tz[l] += (double)acc[l];
            P = Pn;
            G = Gn;
        }
    }
#pragma unroll
    for (int l = 0; l < NH; ++l) {
        const double t = block_sum(tz[l], s_part);
        if (threadIdx.x == 0) atomicAdd(&st->sums[parity].tvz[l0 + l], t);
    }
}

__global__ void __launch_bounds__(kTvThreads) k_tv_apply(float* __restrict__ x, const float* __restrict__ grad, long long n_slots, TvState* st,
                                                  int parity, int n_half, float gamma) {
    const TvSums& sm = st->sums[parity];
    const double g2 = sm.g2, tvx = sm.tvx;
    const float beta = st->beta[parity];
    int level = -1;
    if (g2 > 0.0) {
        for (int l = n_half - 1; l >= 0; --l)
            if (sm.tvz[l] <= tvx) level = l;  // the FIRST level that does not raise the total variation
    }
    float used = beta;
    for (int l = 0; l < (level >= 0 ? level : n_half); ++l) used *= 0.5f;
    if (level >= 0) {
        const float s = used / (float)sqrt(g2);
        const long long stride = (long long)gridDim.x * blockDim.x, n4 = n_slots >> 2;  // (a slice is whole tiles: n_slots % 4 == 0)
        float4* x4 = reinterpret_cast<float4*>(x);
        const float4* g4 = reinterpret_cast<const float4*>(grad);
        for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += stride) {
            float4 v = x4[q];
            const float4 d = g4[q];
            v.x = fmaf(-s, d.x, v.x), v.y = fmaf(-s, d.y, v.y), v.z = fmaf(-s, d.z, v.z), v.w = fmaf(-s, d.w, v.w);
            x4[q] = v;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {  // (fields no thread of this launch reads)
        st->beta[parity ^ 1] = gamma * used;
        st->beta_used = used;
        st->level = level;
        st->tv_before = tvx;
        st->tv_after = level >= 0 ? sm.tvz[level] : tvx;
        st->steps += 1u;
        st->accepted += level >= 0 ? 1u : 0u;
        TvSums& other = st->sums[parity ^ 1];  // the next step's sums (nothing reads them during this step)
        other.tvx = other.g2 = 0.0;
        for (int l = 0; l < kTvMaxLevels; ++l) other.tvz[l] = 0.0;
    }
}

// Chunk of slices per work item: every chunk costs one extra slice (the terms below its first), every round of the grid
// runs as long as its chunk: the smallest rounds x (chunk + 1/2).
static TvItems plan_items(const Geom& g, int warp_slots) {
    TvItems w;
    w.nxt = g.nxp / 2;
    w.nyt = g.slice_p / (2 * g.nxp);
    w.wx_n = (w.nxt + 31) / 32;
    double best = 0.0;
    w.chunk = g.nz;
    for (int c = 1; c <= g.nz; ++c) {
        const long long items = (long long)w.wx_n * w.nyt * ((g.nz + c - 1) / c);
        const double cost = (double)((items + warp_slots - 1) / warp_slots) * (c + 0.5);
        if (best == 0.0 || cost < best) best = cost, w.chunk = c;
    }
    w.n_items = w.wx_n * w.nyt * ((g.nz + w.chunk - 1) / w.chunk);
    return w;
}

cudaError_t launch_tvs_step(float* x, float* grad, const Geom& g, long long n_slots, TvState* st, int parity, int n_half, float gamma,
                            int sms, cudaStream_t stream) {
    typedef void (*probe_fn)(const float*, const float*, Geom, TvItems, TvState*, int, int);
    static const probe_fn probes[kTvMaxLevels] = {k_tv_probe<1>, k_tv_probe<2>, k_tv_probe<3>, k_tv_probe<4>,
                                                  k_tv_probe<5>, k_tv_probe<6>, k_tv_probe<7>, k_tv_probe<8>};
    static int per_sm_grad = 0, per_sm_probe_of[kTvMaxLevels] = {0};
    if (n_half < 1 || n_half > kTvMaxLevels) return cudaErrorInvalidValue;
    if (!per_sm_grad) {
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_grad, k_tv_grad, kTvThreads, 0);
        if (per_sm_grad < 1) per_sm_grad = 1;
        for (int n = 0; n < kTvMaxLevels; ++n) {
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_probe_of[n], probes[n], kTvThreads, 0);
            if (per_sm_probe_of[n] < 1) per_sm_probe_of[n] = 1;
        }
    }
    if (sms <= 0) sms = 148;
    const int wpb = kTvThreads / 32;
    const TvItems wg = plan_items(g, sms * per_sm_grad * wpb);
    const int grid_g = std::min((wg.n_items + wpb - 1) / wpb, sms * per_sm_grad);
    long long blocks = std::min<long long>((n_slots + 4 * kTvThreads - 1) / (4 * kTvThreads), (long long)sms * 8);
    if (blocks < 1) blocks = 1;
    k_tv_grad<<<grid_g, kTvThreads, 0, stream>>>(x, grad, g, wg, st, parity);
    for (int part = 0; part < 2; ++part) {  // level 0, then the others
        const int nh = part == 0 ? 1 : n_half - 1;
        if (nh < 1) break;
        const int per_sm = per_sm_probe_of[nh - 1];
        const TvItems wp = plan_items(g, sms * per_sm * wpb);
        const int grid_p = std::min((wp.n_items + wpb - 1) / wpb, sms * per_sm);
        probes[nh - 1]<<<grid_p, kTvThreads, 0, stream>>>(x, grad, g, wp, st, parity, part);
    }
    k_tv_apply<<<(int)blocks, kTvThreads, 0, stream>>>(x, grad, n_slots, st, parity, n_half, gamma);
    return cudaGetLastError();
}

}  // namespace pct
