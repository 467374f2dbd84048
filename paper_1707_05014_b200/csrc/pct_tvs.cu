// pct_tvs.cu -- total-variation superiorization step on the image ("both
// algorithms incorporate total variation superiorization (TVS), which 'jiggles' the solution ... In CARP, TVS is applied
// just once to the initial solution at the start of each iteration.  In DROP, however, TVS is applied to the initial
// solution that enters each block").  The paper prints no formula; R31 fixes the step:
//
//   TV(x) = sum_ijk sqrt(dx^2 + dy^2 + dz^2 + eps^2)  (forward differences, zero across the far faces, eps = 1e-6)
//   g = grad TV(x);  v = -g / ||g||;  z_l = x + beta 2^-l v, l = 0 .. n_half-1;  x <- the first z_l with TV(z_l) <= TV(x)
//   beta <- gamma * (the step that was taken, or beta 2^-n_half if none was)
//
// Four launches per step, all on the image in its storage order (voxel_slot: 2 x 2 in-plane tiles):
//   k_tv_reset  zeroes the sums;   k_tv_grad  g and the fp64 sums TV(x), ||g||^2;
//   k_tv_probe  TV(z_l) for every level at once (z is never stored: its differences follow from those of x and g);
//   k_tv_apply  picks the level from the sums (every thread, identically) and moves the image.
// Terms are formed in fp32, summed in fp64 (block tree, then one atomic per block): the comparison TV(z) <= TV(x) is
// taken on sums whose rounding is far below the change a step makes.
#include "pct_internal.h"

namespace pct {

constexpr float kTvEps2 = 1.0e-12f;  // eps^2

struct Nb {  // a voxel and its forward differences
    float c, dx, dy, dz;
};

__device__ __forceinline__ float at(const float* __restrict__ a, const Geom& g, int i, int j, int k) {
    return __ldg(a + voxel_slot(i, j, k, g.nxp, g.slice_p));
}

__device__ __forceinline__ Nb forward(const float* __restrict__ a, const Geom& g, int i, int j, int k) {
    Nb n;
    n.c = at(a, g, i, j, k);
    n.dx = i + 1 < g.nx ? at(a, g, i + 1, j, k) - n.c : 0.0f;
    n.dy = j + 1 < g.ny ? at(a, g, i, j + 1, k) - n.c : 0.0f;
    n.dz = k + 1 < g.nz ? at(a, g, i, j, k + 1) - n.c : 0.0f;
    return n;
}

// t = sqrt(q) and 1 / t from one reciprocal square root (relative error 2^-22: far inside the step's tolerance)
__device__ __forceinline__ float rterm(const Nb& n, float& t) {
    const float q = n.dx * n.dx + n.dy * n.dy + n.dz * n.dz + kTvEps2;
    const float r = rsqrtf(q);
    t = q * r;
    return r;
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

__global__ void k_tv_reset(TvState* st) {
    st->tvx = 0.0;
    st->g2 = 0.0;
    for (int l = 0; l < kTvMaxLevels; ++l) st->tvz[l] = 0.0;
}

// Tile rows (one per CTA trip): entry q of tile row jt of a slice is voxel i = 2 (q >> 2) + (q & 1), j = 2 jt + ((q >> 1) & 1)
// (voxel_slot read backwards, no division).
__device__ __forceinline__ void tile_row_voxel(int q, int jt, int& i, int& j) {
    i = ((q >> 2) << 1) + (q & 1);
    j = 2 * jt + ((q >> 1) & 1);
}

__global__ void __launch_bounds__(256) k_tv_grad(const float* __restrict__ x, float* __restrict__ grad, const Geom g, TvState* st) {
    __shared__ double s_part[8];
    double tv = 0.0, g2 = 0.0;
    const int n_jt = g.slice_p / (2 * g.nxp), n_rows = n_jt * g.nz;
    for (int row = blockIdx.x; row < n_rows; row += gridDim.x) {  // (a persistent grid: one block sum per CTA, not per row)
    const int k = row / n_jt, jt = row - k * n_jt;
    const long long row0 = (long long)k * g.slice_p + (long long)jt * 2 * g.nxp;
    for (int q = threadIdx.x; q < 2 * g.nxp; q += blockDim.x) {
        int i, j;
        tile_row_voxel(q, jt, i, j);
        float gv = 0.0f;
        if (i < g.nx && j < g.ny) {  // (padding slots of odd grids hold nothing)
            const Nb n = forward(x, g, i, j, k);
            float t;
            const float r = rterm(n, t);
            gv = -(n.dx + n.dy + n.dz) * r;  // d t_ijk / d x_ijk
            float tm;
            if (i > 0) {                        // + d t_(i-1)jk / d x_ijk, ...
                const Nb m = forward(x, g, i - 1, j, k);
                gv += m.dx * rterm(m, tm);
            }
            if (j > 0) {
                const Nb m = forward(x, g, i, j - 1, k);
                gv += m.dy * rterm(m, tm);
            }
            if (k > 0) {
                const Nb m = forward(x, g, i, j, k - 1);
                gv += m.dz * rterm(m, tm);
            }
            tv += (double)t;
            g2 += (double)gv * (double)gv;
        }
        grad[row0 + q] = gv;
    }
    }
    const double a = block_sum(tv, s_part);
    const double b = block_sum(g2, s_part);
    if (threadIdx.x == 0) {
        atomicAdd(&st->tvx, a);
        atomicAdd(&st->g2, b);
    }
}

__global__ void __launch_bounds__(256) k_tv_probe(const float* __restrict__ x, const float* __restrict__ grad, const Geom g, TvState* st,
                                                  int parity, int n_half) {
    __shared__ double s_part[8];
    const double g2 = st->g2;
    if (!(g2 > 0.0)) return;  // flat image: no direction, no step
    const float s0 = st->beta[parity] / (float)sqrt(g2);  // z = x - s g,  s = beta 2^-l / ||g||
    double tz[kTvMaxLevels];
#pragma unroll
    for (int l = 0; l < kTvMaxLevels; ++l) tz[l] = 0.0;
    const int n_jt = g.slice_p / (2 * g.nxp), n_rows = n_jt * g.nz;
    for (int row = blockIdx.x; row < n_rows; row += gridDim.x) {
    const int k = row / n_jt, jt = row - k * n_jt;
    for (int q = threadIdx.x; q < 2 * g.nxp; q += blockDim.x) {
        int i, j;
        tile_row_voxel(q, jt, i, j);
        if (i >= g.nx || j >= g.ny) continue;
        const Nb a = forward(x, g, i, j, k), b = forward(grad, g, i, j, k);
        float sl = s0;
#pragma unroll
        for (int l = 0; l < kTvMaxLevels; ++l) {
            if (l < n_half) {
                const float dx = a.dx - sl * b.dx, dy = a.dy - sl * b.dy, dz = a.dz - sl * b.dz;
                const float q2 = dx * dx + dy * dy + dz * dz + kTvEps2;
                tz[l] += (double)(q2 * rsqrtf(q2));
                sl *= 0.5f;
            }
        }
    }
    }
    for (int l = 0; l < n_half; ++l) {
        const double t = block_sum(tz[l], s_part);
        if (threadIdx.x == 0) atomicAdd(&st->tvz[l], t);
    }
}

__global__ void __launch_bounds__(256) k_tv_apply(float* __restrict__ x, const float* __restrict__ grad, long long n_slots, TvState* st,
                                                  int parity, int n_half, float gamma) {
    const double g2 = st->g2, tvx = st->tvx;
    const float beta = st->beta[parity];
    int level = -1;
    if (g2 > 0.0) {
        for (int l = n_half - 1; l >= 0; --l)
            if (st->tvz[l] <= tvx) level = l;  // the FIRST level that does not raise the total variation
    }
    float used = beta;
    for (int l = 0; l < (level >= 0 ? level : n_half); ++l) used *= 0.5f;
    if (level >= 0) {
        const float s = used / (float)sqrt(g2);
        const long long stride = (long long)gridDim.x * blockDim.x;
        for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n_slots; q += stride) x[q] = fmaf(-s, grad[q], x[q]);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {  // (fields no thread of this launch reads)
        st->beta[parity ^ 1] = gamma * used;
        st->beta_used = used;
        st->level = level;
        st->tv_before = tvx;
        st->tv_after = level >= 0 ? st->tvz[level] : tvx;
        st->steps += 1u;
        st->accepted += level >= 0 ? 1u : 0u;
    }
}

cudaError_t launch_tvs_step(float* x, float* grad, const Geom& g, long long n_slots, TvState* st, int parity, int n_half, float gamma,
                            int sms, cudaStream_t stream) {
    long long blocks = (n_slots + 255) / 256;
    const long long cap = (long long)(sms > 0 ? sms : 148) * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    long long rows = (long long)(g.slice_p / (2 * g.nxp)) * g.nz;  // tile rows of the volume, dealt out to a persistent grid
    if (rows > cap) rows = cap;
    k_tv_reset<<<1, 1, 0, stream>>>(st);
    k_tv_grad<<<(int)rows, 256, 0, stream>>>(x, grad, g, st);
    k_tv_probe<<<(int)rows, 256, 0, stream>>>(x, grad, g, st, parity, n_half);
    k_tv_apply<<<(int)blocks, 256, 0, stream>>>(x, grad, n_slots, st, parity, n_half, gamma);
    return cudaGetLastError();
}

}  // namespace pct
