// pct_wave.cu -- the WAVEFRONT engine of the DROP sweep (k_plan_blocks, k_wave).
//
// PAPER.md:50 makes the blocks of a sweep sequential: "The solution x1 is then used as the initial solution for
// the next block".  What a row of block q+1 needs is the image after block q ON THE VOXELS IT TOUCHES, and a
// proton path stays within a few slices of the image (slopes of milliradians): the dependency between two
// consecutive blocks is local in depth.  So:
//
//   k_plan_blocks  once per (histories, block size): for every history the range [sa, sb] of DEPTH SLABS its path
//                  can touch (a rigorous bound from the hull points and the path's shape functions, checked again
//                  by the walk), every block counting-sorted by sa, and need[q][s] = number of histories of block q
//                  whose range holds slab s.
//   k_wave         ONE persistent launch for a whole range of blocks.  Work items (a few histories, consecutive in
//                  the plan's order) are drawn from one ticket counter, block after block.  A warp walks a history
//                  (hull, MLP, voxel walk: nothing of that reads the image), then waits until its slabs hold the
//                  image after the previous block (upd_seq[s] >= q), gathers, scatters.  When the last history
//                  that can touch slab s of block q has scattered (done[q][s] == need[q][s]), the update
//                  x_j += lambda Delta_j / max(1, c_j) of that slab is posted as n_sub sub-tasks which the warps
//                  pick up between histories; the last one to finish publishes upd_seq[s] = q + 1.
//
// The block boundary is therefore a per-slab flag, not a grid-wide barrier: no launch per block, no tail of idle
// warps, no separate sweep of the update kernel over image and accumulator (a slab is updated while it is hot in
// the L2), and the histories of a block are taken slab by slab, so gather and reductions work on a fraction of
// image + accumulator at a time.  The result is DROP's, block for block: every row of block q sees, on every voxel
// of its row, the image after block q-1 (rounding order of the atomic sums aside, R20).
//
// Forward progress: a warp holding ticket w waits only for work of tickets < w (held by resident warps, which never
// wait for a later ticket) and for update sub-tasks, which every waiting warp executes itself.  Every wait is
// bounded: it gives up after a few seconds, sets ctrl->error and the call reports PCT_EINTERNAL.
#include "pct_walk.cuh"

namespace pct {

#ifndef PCT_WAVE_ACQUIRE_PREFETCH
#define PCT_WAVE_ACQUIRE_PREFETCH 1  // the flag load issued before the walk is ld.acquire (0: relaxed)
#endif

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---- slab range of one history (plan) ---------------------------------------------------------------------
// v(s) = v0 + sig_v s + c0(s) be0 + c2(s) be2 on [0, L] (rule step 3c) with shape functions that depend on (s, L)
// only: |c0| <= 0.25 L for L <= 300 mm and <= 0.6 L beyond, |c2| <= 0.16 L (tests/test_wave_plan.py pins both
// against the fp64 matrix form; the spline's are 4/27 L).  The chord part lies between v0 and v2, segment
// midpoints lie between nodes.  margin: fp32 rounding of the node arithmetic (<= 1e-4 mm) and of the
// expressions below.  The walk checks every voxel of every row against the range declared here (gather_row_cg).
__device__ __forceinline__ void slab_range(const Geom& g, const PathState& st, int slab_slices, int n_slabs, int& sa, int& sb) {
    const float k0 = st.L <= 300.0f ? 0.25f : 0.6f;
    const float dev = (k0 * fabsf(st.be0) + 0.16f * fabsf(st.be2)) * st.L;
    const float margin = 0.02f + 1e-5f * g.zmax;
    const float vlo = fminf(st.v0, st.v2) - dev - margin, vhi = fmaxf(st.v0, st.v2) + dev + margin;
    float zl = floorf(vlo * g.inv_h + g.hz), zh = floorf(vhi * g.inv_h + g.hz);
    zl = fminf(fmaxf(zl, 0.0f), g.fnz - 1.0f);
    zh = fminf(fmaxf(zh, 0.0f), g.fnz - 1.0f);
    sa = (int)zl / slab_slices;
    sb = (int)zh / slab_slices;
    if (sb - sa >= 7) {  // (the width code has three bits: 7 = every slab)
        sa = 0;
        sb = n_slabs - 1;
    }
}
constexpr uint32_t kPlanEmpty = (31u << 24) | (7u << 29);  // skipped history: no slab, nothing to wait for or to signal

__device__ __forceinline__ uint32_t plan_code(const HistPtrs& H, const Geom& g, int slab_slices, int n_slabs, long long i, int& sa, int& sb) {
    const Hist hh = load_history(H, i);
    PathState st;
    setup_history(g, hh, st);
    if (st.K < 0) {
        sa = 1;
        sb = 0;
        return kPlanEmpty;
    }
    slab_range(g, st, slab_slices, n_slabs, sa, sb);
    const int w = (sa == 0 && sb == n_slabs - 1 && n_slabs > 7) ? 7 : sb - sa;
    return ((uint32_t)sa << 24) | ((uint32_t)w << 29);
}

__device__ __forceinline__ void plan_decode(uint32_t code, int n_slabs, int& sa, int& sb) {
    sa = (int)((code >> 24) & 31u);
    const int w = (int)(code >> 29);
    if (w == 7) {
        if (sa == 31) {  // kPlanEmpty
            sa = 1;
            sb = 0;
        } else {
            sa = 0;
            sb = n_slabs - 1;
        }
    } else {
        sb = sa + w;
    }
}

__global__ void __launch_bounds__(512) k_plan_blocks(const HistPtrs H, const Geom g, long long n, long long block_size, long long first_block,
                                                     long long n_blocks, int n_slabs, int slab_slices, uint32_t* __restrict__ plan,
                                                     int* __restrict__ need) {
    __shared__ unsigned bins[kMaxSlabs];
    __shared__ unsigned cnts[kMaxSlabs];
    for (long long b = first_block + blockIdx.x; b < first_block + n_blocks; b += gridDim.x) {
        const long long first = b * block_size;
        const long long count = n - first < block_size ? n - first : block_size;
        if (threadIdx.x < kMaxSlabs) bins[threadIdx.x] = cnts[threadIdx.x] = 0u;
        __syncthreads();
        for (long long r = threadIdx.x; r < count; r += blockDim.x) {
            int sa, sb;
            plan_code(H, g, slab_slices, n_slabs, first + r, sa, sb);
            atomicAdd(&bins[sa <= sb ? sa : 0], 1u);
            for (int s = sa; s <= sb; ++s) atomicAdd(&cnts[s], 1u);
        }
        __syncthreads();
        if (threadIdx.x < 32) {  // exclusive scan of the bin counts (kMaxSlabs == 32: one warp)
            const unsigned c = bins[threadIdx.x];
            unsigned incl = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned up = __shfl_up_sync(0xffffffffu, incl, o);
                if ((int)threadIdx.x >= o) incl += up;
            }
            bins[threadIdx.x] = incl - c;
            if ((int)threadIdx.x < n_slabs) need[b * n_slabs + threadIdx.x] = (int)cnts[threadIdx.x];
        }
        __syncthreads();
        for (long long r = threadIdx.x; r < count; r += blockDim.x) {
            int sa, sb;
            const uint32_t code = plan_code(H, g, slab_slices, n_slabs, first + r, sa, sb);
            const unsigned pos = atomicAdd(&bins[sa <= sb ? sa : 0], 1u);
            plan[first + pos] = code | (uint32_t)r;
        }
        __syncthreads();
    }
}

// ---- update sub-tasks -------------------------------------------------------------------------------------

__device__ __forceinline__ float updated_w(float xv, float d, float c, float lambda) {
    return c > 0.0f ? xv + __fdiv_rn(lambda * d, c) : xv;
}

// x_j += lambda Delta_j / max(1, c_j) on sub-task `sub` of slab s (R12); the accumulator entries that were hit are
// zeroed.  Image and accumulator are read past the L1 (the reductions of other SMs live in the L2).
__device__ __forceinline__ void update_subtask(const WaveArgs& a, int s, int sub, int lane) {
    const long long v0 = (long long)s * a.slab_voxels;
    const long long v1 = v0 + a.slab_voxels < a.n_voxels ? v0 + a.slab_voxels : a.n_voxels;
    if ((a.slab_voxels & 3) == 0) {
        const long long n4 = (v1 - v0) >> 2;  // (v1 - v0 is a multiple of four: whole slices of nx*ny voxels, nx*ny*slab_slices % 4 == 0)
        const long long per = (n4 + a.n_sub - 1) / a.n_sub;
        const long long g0 = (v0 >> 2) + (long long)sub * per;
        const long long g1 = g0 + per < (v0 >> 2) + n4 ? g0 + per : (v0 >> 2) + n4;
        float4* x4 = reinterpret_cast<float4*>(a.x);
        float4* a4 = reinterpret_cast<float4*>(a.acc);
        constexpr int UN = 4;
        for (long long q0 = g0 + lane; q0 < g1; q0 += 32 * UN) {
            float4 a01[UN], a23[UN], xv[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const long long q = q0 + 32 * u;
                if (q < g1) {
                    a01[u] = __ldcg(a4 + 2 * q);
                    a23[u] = __ldcg(a4 + 2 * q + 1);
                    xv[u] = __ldcg(x4 + q);
                } else {
                    a01[u] = a23[u] = xv[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const long long q = q0 + 32 * u;
                const bool hit01 = a01[u].y > 0.0f || a01[u].w > 0.0f, hit23 = a23[u].y > 0.0f || a23[u].w > 0.0f;
                if (hit01 || hit23) {
                    float4 v = xv[u];
                    v.x = updated_w(v.x, a01[u].x, a01[u].y, a.lambda);
                    v.y = updated_w(v.y, a01[u].z, a01[u].w, a.lambda);
                    v.z = updated_w(v.z, a23[u].x, a23[u].y, a.lambda);
                    v.w = updated_w(v.w, a23[u].z, a23[u].w, a.lambda);
                    __stcg(x4 + q, v);
                    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (hit01) __stcg(a4 + 2 * q, z);
                    if (hit23) __stcg(a4 + 2 * q + 1, z);
                }
            }
        }
    } else {  // grids whose slabs are not a multiple of four voxels: one voxel at a time
        const long long nv = v1 - v0;
        const long long per = (nv + a.n_sub - 1) / a.n_sub;
        const long long j0 = v0 + (long long)sub * per;
        const long long j1 = j0 + per < v1 ? j0 + per : v1;
        for (long long j = j0 + lane; j < j1; j += 32) {
            const float2 dc = __ldcg(a.acc + j);
            if (dc.y > 0.0f) {
                __stcg(a.x + j, updated_w(__ldcg(a.x + j), dc.x, dc.y, a.lambda));
                __stcg(a.acc + j, make_float2(0.f, 0.f));
            }
        }
    }
}

// Claim and run one posted update sub-task, if there is one.  Warp-collective.  Returns false iff none was found.
__device__ __forceinline__ bool try_update(const WaveArgs& a, int lane, unsigned warp_id) {
    WaveCtrl* c = a.ctrl;
    unsigned p = 0, cl = 0;
    if (lane < a.n_slabs) {
        p = ld_acquire_u32(&c->posted[lane]);
        cl = ld_relaxed_u32(&c->claimed[lane]);
    }
    const unsigned avail = __ballot_sync(0xffffffffu, cl < p * (unsigned)a.n_sub);
    if (avail == 0u) return false;
    // the warps spread over the slabs that have work: first available slab at or after a warp-dependent start
    const unsigned rot = warp_id & 31u;
    const unsigned hi = avail >> rot;
    const int s = hi ? (int)rot + __ffs(hi) - 1 : __ffs(avail) - 1;
    const unsigned mine = __shfl_sync(0xffffffffu, cl, s);
    int got = 0;
    if (lane == 0) {
        got = atomicCAS(&c->claimed[s], mine, mine + 1u) == mine;
        if (got) atomicSub(&c->pending, 1);
    }
    got = __shfl_sync(0xffffffffu, got, 0);
    if (!got) return true;  // another warp took it; there may be more
    const unsigned seq = ld_relaxed_u32(&c->post_seq[s]);  // (written before `posted` moved: ordered by the acquire above)
    update_subtask(a, s, (int)(mine % (unsigned)a.n_sub), lane);
    __threadfence();  // every lane's stores, before the counter moves
    __syncwarp();
    if (lane == 0) {
        const unsigned f = atomicAdd(&c->finished[s], 1u);
        if ((f + 1u) % (unsigned)a.n_sub == 0u) {  // the last sub-task of this update
            __threadfence();
            st_release_u32(&c->upd_seq[s], seq + 1u);
        }
    }
    return true;
}

// The update of slab s after block q is due: post its sub-tasks.
__device__ __forceinline__ void post_update(const WaveArgs& a, int s, unsigned q) {
    WaveCtrl* c = a.ctrl;
    __threadfence();  // (acquire side of the done[] counter: the other warps' reductions are ordered before what follows)
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(&c->post_seq[s]), "r"(q) : "memory");
    __threadfence();
    atomicAdd(&c->posted[s], 1u);
    atomicAdd(&c->pending, a.n_sub);
}

constexpr unsigned kSpinLimit = 1u << 23;  // x >= 100 ns: a wait gives up after about a second of doing nothing

// Wait until slabs [sa, sb] hold the image after blocks [0, q) of the sweep.  Lane l looks after slab sa + l; `flag` is
// the value of upd_seq it loaded before the walk.  A block without a history for a slab never posts an update for
// it: whoever waits moves upd_seq over such blocks (need == 0) itself.  While waiting the warp runs update sub-tasks.
__device__ __forceinline__ bool wait_slabs(const WaveArgs& a, int lane, unsigned warp_id, int sa, int sb, unsigned q, unsigned flag) {
    WaveCtrl* c = a.ctrl;
    const bool mine = lane <= sb - sa;
    bool ok = !mine || flag >= q;
    if (__all_sync(0xffffffffu, ok)) return true;
    unsigned spins = 0;
    for (;;) {
        if (!ok) {
            const int s = sa + lane;
            unsigned u = ld_acquire_u32(&c->upd_seq[s]);
            if (u < q && __ldg(a.need + (long long)u * a.n_slabs + s) == 0) {
                atomicCAS(&c->upd_seq[s], u, u + 1u);  // block u has nothing for this slab
                u = ld_acquire_u32(&c->upd_seq[s]);
            }
            ok = u >= q;
        }
        if (__all_sync(0xffffffffu, ok)) return true;
        if (!try_update(a, lane, warp_id)) {
            __nanosleep(100);
            unsigned err = 0;
            if (lane == 0) err = ld_relaxed_u32(&c->error) & 2u;
            err = __shfl_sync(0xffffffffu, err, 0);
            if (++spins > kSpinLimit || err) {
                if (lane == 0) atomicOr(&c->error, 2u);
                return false;
            }
        }
    }
}

template <bool SPLINE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) k_wave(const WaveArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned warp_id = blockIdx.x * kWarpsPerCta + warp;
    const SmemLayout lay = smem_layout(g.nmin);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * lay.row_slots;
    stage_table(s_tab, a.tab, g.nmin);
    WaveCtrl* ctrl = a.ctrl;
    const bool planned = a.plan != nullptr;
    const long long B = planned ? a.block_size : a.count;
    const long long ipb = (B + a.item - 1) / a.item;  // items per block
    const unsigned long long n_items = planned ? (unsigned long long)(a.q1 - a.q0) * ipb : (unsigned long long)ipb;
    unsigned long long rows = 0, nnz_total = 0, segs = 0;
    const EmitPtrs no_emit{nullptr, nullptr, nullptr, nullptr};
    bool give_up = false;

    while (!give_up) {
        if (planned) {  // posted updates first: other warps wait for them
            int pend = 0;
            if (lane == 0) pend = (int)ld_relaxed_u32(reinterpret_cast<const unsigned*>(&ctrl->pending));
            pend = __shfl_sync(0xffffffffu, pend, 0);
            while (pend > 0 && try_update(a, lane, warp_id)) {
                if (lane == 0) pend = (int)ld_relaxed_u32(reinterpret_cast<const unsigned*>(&ctrl->pending));
                pend = __shfl_sync(0xffffffffu, pend, 0);
            }
        }
        unsigned long long w = 0;
        if (lane == 0) w = atomicAdd(&ctrl->ticket, 1ULL);
        w = __shfl_sync(0xffffffffu, w, 0);
        if (w >= n_items) break;
        const long long q = planned ? a.q0 + (long long)(w / (unsigned long long)ipb) : 0;  // block of the sweep
        const long long rel0 = (long long)(w % (unsigned long long)ipb) * a.item;
        const long long first = planned ? q * a.block_size : a.first;
        const long long count = planned ? (a.n - first < a.block_size ? a.n - first : a.block_size) : a.count;
        const int cnt = count - rel0 < a.item ? (int)(count - rel0) : a.item;
        if (cnt <= 0) continue;  // (the short last block has fewer items)
        int my_sa = 1, my_sb = 0;  // slab range of the history this lane sets up
        if (lane < cnt) {
            long long r = rel0 + lane;
            if (planned) {
                const uint32_t code = __ldg(a.plan + first + r);
                r = (long long)(code & 0xffffffu);
                plan_decode(code, a.n_slabs, my_sa, my_sb);
            }
            const Hist hh = load_history(a.H, first + r);
            setup_history(g, hh, s_state[lane]);
        }
        __syncwarp();
        for (int p = 0; p < cnt && !give_up; ++p) {
            const PathState& S = s_state[p];
            const int K = S.K;
            if (K < 0) continue;  // skipped history: empty row (R7)
            const int sa = __shfl_sync(0xffffffffu, my_sa, p), sb = __shfl_sync(0xffffffffu, my_sb, p);
            unsigned flag = 0xffffffffu;
            if (planned && lane <= sb - sa) {
#if PCT_WAVE_ACQUIRE_PREFETCH
                flag = ld_acquire_u32(&ctrl->upd_seq[sa + lane]);
#else
                flag = ld_relaxed_u32(&ctrl->upd_seq[sa + lane]);
#endif
            }
            float nrm;
            int nnz;
            walk_history<false, SPLINE>(g, S, s_tab, lane, row, nrm, nnz, no_emit);
            const int C = (K + 32) >> 5;
            unsigned lo = 0u, span = 0xffffffffu;
            if (planned) {
                if (!wait_slabs(a, lane, warp_id, sa, sb, (unsigned)q, flag)) {
                    give_up = true;
                    break;
                }
                lo = (unsigned)((long long)sa * a.slab_voxels);
                span = (unsigned)((long long)(sb - sa + 1) * a.slab_voxels);
            }
            bool bad = false;
            float dot = gather_row_cg(row, lane, C, a.x, lo, span, bad);
            dot = warp_sum(dot);
            nrm = warp_sum(nrm);
            if (__any_sync(0xffffffffu, bad)) {  // the plan's range does not hold the row: never scatter outside it
                if (lane == 0) atomicOr(&ctrl->error, 1u);
            } else if (nrm > 0.0f) {  // non-empty row (R13)
                const float r = __fdiv_rn(S.wepl - dot, nrm);
                scatter_row(row, lane, C, a.acc, r);
                rows += (lane == 0);
                nnz_total += nnz;
            }
            __syncwarp();  // the row buffer is reused by the next history
            segs += (lane == 0) ? (K + 1) : 0;
            if (planned && p + 1 < cnt) {  // an update posted meanwhile? (one load per history)
                int pend = 0;
                if (lane == 0) pend = (int)ld_relaxed_u32(reinterpret_cast<const unsigned*>(&ctrl->pending));
                pend = __shfl_sync(0xffffffffu, pend, 0);
                if (pend > 0) try_update(a, lane, warp_id);
            }
        }
        if (planned) {
            // the item has scattered: every lane's reductions are ordered before the counters move
            __threadfence();
            __syncwarp();
            int mine = 0;  // histories of the item whose range holds slab `lane`
            for (int p = 0; p < cnt; ++p) {
                const int sa = __shfl_sync(0xffffffffu, my_sa, p), sb = __shfl_sync(0xffffffffu, my_sb, p);
                mine += (lane >= sa && lane <= sb) ? 1 : 0;
            }
            if (mine > 0 && !give_up) {
                const long long slot = q * a.n_slabs + lane;
                const int old = atomicAdd(a.done + slot, mine);
                if (old + mine == __ldg(a.need + slot)) post_update(a, lane, (unsigned)q);
            }
        }
        __syncwarp();  // the state records are reused by the next item
    }
    if (planned && !give_up) {
        // no work left to draw: run update sub-tasks until every slab holds the image after block q1 - 1
        wait_slabs(a, lane, warp_id, 0, a.n_slabs - 1, (unsigned)a.q1, 0u);
    }
    nnz_total = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)nnz_total);
    if (lane == 0) {
        atomicAdd(&ctrl->cur[0], rows);
        atomicAdd(&ctrl->cur[1], nnz_total);
        atomicAdd(&ctrl->cur[2], segs);
    }
}

WaveShape wave_shape(const Geom& g) {
    WaveShape s;
    // slabs of at least 4 mm (a typical path spans a millimetre or two in depth) and at most kMaxSlabs of them
    int by_count = (g.nz + kMaxSlabs - 1) / kMaxSlabs;
    int by_mm = (int)(4.0f / g.h + 0.999f);
    s.slab_slices = by_count > by_mm ? by_count : by_mm;
    if (s.slab_slices < 1) s.slab_slices = 1;
    if (s.slab_slices > g.nz) s.slab_slices = g.nz;
    s.n_slabs = (g.nz + s.slab_slices - 1) / s.slab_slices;
    // sub-tasks of about 2048 groups of four voxels (64 per lane)
    const long long groups = (long long)s.slab_slices * g.nx * g.ny / 4;
    long long ns = (groups + 2047) / 2048;
    s.n_sub = ns < 1 ? 1 : (ns > 256 ? 256 : (int)ns);
    return s;
}

cudaError_t wave_configure(int nmin, int* grid_out) {
    if (((nmin + 32) >> 5) > 64) return cudaErrorInvalidValue;
    const size_t smem = drop_smem_bytes(nmin);
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_wave<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_wave<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_wave<false>, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    *grid_out = sms * per_sm;
    return cudaSuccess;
}

cudaError_t launch_wave(const WaveArgs& a, int grid, cudaStream_t stream) {
    // never more warps than items
    const long long B = a.plan ? a.block_size : a.count;
    const long long ipb = (B + a.item - 1) / a.item;
    const long long items = a.plan ? (a.q1 - a.q0) * ipb : ipb;
    const long long need = (items + kWarpsPerCta - 1) / kWarpsPerCta;
    if (need < grid) grid = need < 1 ? 1 : (int)need;
    const size_t smem = drop_smem_bytes(a.g.nmin);
    if (a.g.path_model == 1)
        k_wave<true><<<grid, kThreads, smem, stream>>>(a);
    else
        k_wave<false><<<grid, kThreads, smem, stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_plan_blocks(const HistPtrs& H, const Geom& g, long long n, long long block_size, long long first_block,
                               long long n_blocks, const WaveShape& shp, uint32_t* plan, int* need, cudaStream_t stream) {
    if (n_blocks < 1) return cudaSuccess;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long grid = n_blocks < (long long)sms * 4 ? n_blocks : (long long)sms * 4;
    k_plan_blocks<<<(int)grid, 512, 0, stream>>>(H, g, n, block_size, first_block, n_blocks, shp.n_slabs, shp.slab_slices, plan, need);
    return cudaGetLastError();
}

}  // namespace pct
