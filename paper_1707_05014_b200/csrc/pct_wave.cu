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
#include <stdio.h>
#include <string.h>

#include "pct_walk.cuh"

namespace pct {

// Build with -DPCT_WAVE_PROF to accumulate, per phase of k_wave, the cycles its warps spent there (a tuning aid:
// wave_prof_dump prints and clears the totals); the default build carries none of it.
#ifdef PCT_WAVE_PROF
__device__ unsigned long long g_wave_prof[16];
#define PROF_DECL long long prof_t = clock64(); unsigned long long prof_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}
#define PROF(i) do { const long long now__ = clock64(); prof_acc[i] += (unsigned long long)(now__ - prof_t); prof_t = now__; } while (0)
#define PROF_FLUSH do { if (lane == 0) for (int i__ = 0; i__ < 8; ++i__) atomicAdd(&g_wave_prof[i__], prof_acc[i__]); } while (0)
#define UPROF(i) do { if (stage != nullptr) { const long long now__ = clock64(); if (lane == 0) atomicAdd(&g_wave_prof[8 + (i)], (unsigned long long)(now__ - uprof_t)); uprof_t = now__; } } while (0)
#define UPROF_DECL long long uprof_t = clock64()
#define UPROF_COUNT(i) do { if (stage != nullptr && lane == 0) atomicAdd(&g_wave_prof[8 + (i)], 1ULL); } while (0)
#else
#define PROF_DECL
#define PROF(i)
#define PROF_FLUSH
#define UPROF(i)
#define UPROF_DECL
#define UPROF_COUNT(i)
#endif

// Warp roles.  The first kWalkers warps of a CTA walk histories; the last kUpdaters warps only run posted update
// sub-tasks, staged through shared memory with cp.async so that a whole sub-task is ONE memory round trip: an update
// must be finished long before the next block reaches its slab, and a walker's registers are taken by the walk.
#ifndef PCT_WAVE_UPDATERS
#define PCT_WAVE_UPDATERS 2
#endif
constexpr int kUpdaters = PCT_WAVE_UPDATERS;
constexpr int kWalkers = kWarpsPerCta - kUpdaters;
constexpr int kStageGroups = 256;                // groups of four voxels staged at once by an updater warp
constexpr int kStageBytes = kStageGroups * 48;   // 32 B of accumulator + 16 B of image per group
static_assert(kUpdaters >= 0 && kWalkers >= 1, "a CTA needs walkers");  // (kUpdaters = 0: the walkers run the updates while they wait)

__host__ __device__ inline int wave_stage_off(int nmin) { return (smem_layout(nmin).total + 15) & ~15; }
static size_t wave_smem_bytes(int nmin) { return (size_t)wave_stage_off(nmin) + (size_t)kUpdaters * kStageBytes; }

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
    if ((a.g.slice_p & 3) == 0) {  // (always: stored slices have even sides) 128 bits at a time
        const long long n4 = (v1 - v0) >> 2;
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

// The same sub-task by an updater warp: accumulator and image of up to kStageGroups groups go to shared memory with
// cp.async (L2 only, no registers: the whole chunk is in flight at once), are combined there and written back.
__device__ __forceinline__ void update_subtask_staged(const WaveArgs& a, int s, int sub, int lane, float4* stage) {
    const long long v0 = (long long)s * a.slab_voxels;
    const long long v1 = v0 + a.slab_voxels < a.n_voxels ? v0 + a.slab_voxels : a.n_voxels;
    const long long n4 = (v1 - v0) >> 2;
    const long long per = (n4 + a.n_sub - 1) / a.n_sub;
    const long long g0 = (v0 >> 2) + (long long)sub * per;
    const long long g1 = g0 + per < (v0 >> 2) + n4 ? g0 + per : (v0 >> 2) + n4;
    float4* x4 = reinterpret_cast<float4*>(a.x);
    float4* a4 = reinterpret_cast<float4*>(a.acc);
    float4* s_acc = stage;
    float4* s_x = stage + 2 * kStageGroups;
    const unsigned sa_acc = (unsigned)__cvta_generic_to_shared(s_acc), sa_x = (unsigned)__cvta_generic_to_shared(s_x);
    for (long long c0 = g0; c0 < g1; c0 += kStageGroups) {
        const int ng = g1 - c0 < kStageGroups ? (int)(g1 - c0) : kStageGroups;
        const float4* ga = a4 + 2 * c0;
        const float4* gx = x4 + c0;
        for (int i = lane; i < 2 * ng; i += 32)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa_acc + 16u * (unsigned)i), "l"(ga + i) : "memory");
        for (int i = lane; i < ng; i += 32)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa_x + 16u * (unsigned)i), "l"(gx + i) : "memory");
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
        __syncwarp();
        for (int i = lane; i < ng; i += 32) {
            const float4 a01 = s_acc[2 * i], a23 = s_acc[2 * i + 1];
            const bool hit01 = a01.y > 0.0f || a01.w > 0.0f, hit23 = a23.y > 0.0f || a23.w > 0.0f;
            if (hit01 || hit23) {
                float4 v = s_x[i];
                v.x = updated_w(v.x, a01.x, a01.y, a.lambda);
                v.y = updated_w(v.y, a01.z, a01.w, a.lambda);
                v.z = updated_w(v.z, a23.x, a23.y, a.lambda);
                v.w = updated_w(v.w, a23.z, a23.w, a.lambda);
                __stcg(x4 + c0 + i, v);
                const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
                if (hit01) __stcg(a4 + 2 * (c0 + i), z);
                if (hit23) __stcg(a4 + 2 * (c0 + i) + 1, z);
            }
        }
        __syncwarp();  // the staging buffer is overwritten by the next chunk
    }
}

__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acq_rel() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }

__device__ __forceinline__ bool task_open(unsigned long long t) { return (unsigned)(t >> 32) < (unsigned)t; }  // claimed < posted

// Run sub-task `sub` of the update of slab s that was posted last, then count it; the last one of the update
// publishes upd_seq.  Warp-collective.
__device__ __noinline__ void run_update(const WaveArgs& a, int s, unsigned sub, int lane, float4* stage) {
    WaveCtrl* c = a.ctrl;
    // (no fence on this side of the claim: the CAS that won it returned before anything below is issued, and what
    // follows reads the L2, where post_seq and every reduction of the block were visible before the post)
    UPROF_DECL;
    const unsigned seq = ld_relaxed_u32(&c->post_seq[s]);
    if (stage != nullptr && (a.g.slice_p & 3) == 0)
        update_subtask_staged(a, s, (int)sub, lane, stage);
    else
        update_subtask(a, s, (int)sub, lane);
    UPROF(1);
    fence_acq_rel();  // every lane's stores, before the counter moves
    __syncwarp();
    UPROF(2);
    UPROF_COUNT(5);
    if (lane == 0) {
        const unsigned f = atomicAdd(&c->finished[s], 1u);
        if ((f + 1u) % (unsigned)a.n_sub == 0u) {  // the last sub-task of this update
            fence_acq_rel();
            st_release_u32(&c->upd_seq[s], seq + 1u);
        }
    }
}

// Claim one sub-task of slab s given the task word `t` just read (claimed < posted).  One attempt: a warp that loses
// the race goes back to its histories (somebody else is at it).  Warp-collective; returns true iff a sub-task was run.
__device__ __forceinline__ bool claim_and_run(const WaveArgs& a, int s, unsigned long long t, int lane, float4* stage) {
    int got = 0;
    if (lane == 0) {
        // the poster may add to the low half between the load and the CAS: retry once with what the CAS returned
        unsigned long long seen = atomicCAS(&a.ctrl->tasks[s], t, t + (1ULL << 32));
        got = seen == t;
        if (!got && (seen >> 32) == (t >> 32) && task_open(seen)) {
            t = seen;
            got = atomicCAS(&a.ctrl->tasks[s], t, t + (1ULL << 32)) == t;
        }
    }
    got = __shfl_sync(0xffffffffu, got, 0);
    if (!got) return false;
    run_update(a, s, (unsigned)(t >> 32) % (unsigned)a.n_sub, lane, stage);
    return true;
}

// Look at EVERY slab for an open update sub-task and run one (used where the warp has nothing better to do: while it
// waits for a slab, and after the last work item).  Warp-collective.  Returns false iff nothing was open.
__device__ __noinline__ bool steal_update(const WaveArgs& a, int lane, unsigned warp_id, float4* stage) {
    unsigned long long t = 0;
    if (lane < a.n_slabs) t = ld_relaxed_u64(&a.ctrl->tasks[lane]);
    const unsigned avail = __ballot_sync(0xffffffffu, task_open(t));
    if (avail == 0u) return false;
    const unsigned rot = warp_id & 31u;  // the warps spread over the slabs that have work
    const unsigned hi = avail >> rot;
    const int s = hi ? (int)rot + __ffs(hi) - 1 : __ffs(avail) - 1;
    t = __shfl_sync(0xffffffffu, t, s);
    claim_and_run(a, s, t, lane, stage);
    return true;
}

// The update of slab s after block q is due: post its sub-tasks.
__device__ __forceinline__ void post_update(const WaveArgs& a, int s, unsigned q) {
    WaveCtrl* c = a.ctrl;
    fence_acq_rel();  // (acquire side of the done[] counter: the other warps' reductions are ordered before what follows)
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(&c->post_seq[s]), "r"(q) : "memory");
    fence_acq_rel();
    atomicAdd(&c->tasks[s], (unsigned long long)a.n_sub);
}

constexpr unsigned kSpinLimit = 1u << 20;  // x 2-4 us: a wait gives up after a few seconds of doing nothing

// Do slabs [sa, sb] hold the image after blocks [0, q) of the sweep?  Lane l looks after slab sa + l (`ok` carries its
// answer from call to call).  A block without a history for a slab never posts an update for it: whoever asks moves
// upd_seq over such blocks (need == 0) itself.  Warp-collective.
__device__ __forceinline__ bool slabs_reached(const WaveArgs& a, int lane, int sa, int sb, unsigned q, bool& ok) {
    WaveCtrl* c = a.ctrl;
    if (!ok && lane <= sb - sa) {
        const int s = sa + lane;
        unsigned u = ld_acquire_u32(&c->upd_seq[s]);
        while (u < q && __ldg(a.need + (long long)u * a.n_slabs + s) == 0) {
            atomicCAS(&c->upd_seq[s], u, u + 1u);  // block u has nothing for this slab
            u = ld_acquire_u32(&c->upd_seq[s]);
        }
        ok = u >= q;
    }
    return __all_sync(0xffffffffu, ok || lane > sb - sa);
}

__device__ __forceinline__ bool wave_failed(WaveCtrl* c, int lane) {
    unsigned err = 0;
    if (lane == 0) err = ld_relaxed_u32(&c->error) & 2u;
    return __shfl_sync(0xffffffffu, err, 0) != 0u;
}

// A walker waits for the slabs of the history it has just walked.  The updater warps do the updates; a walker that
// has waited for a while lends a hand (register path), which also keeps the launch alive whatever is resident.
__device__ __noinline__ bool wait_slabs_slow(const WaveArgs& a, int lane, unsigned warp_id, int sa, int sb, unsigned q) {
    bool ok = false;
    for (unsigned spins = 0;; ++spins) {
        if (slabs_reached(a, lane, sa, sb, q, ok)) return true;
        if (spins >= 8u && steal_update(a, lane, warp_id, nullptr)) continue;
        // back off: thousands of warps may wait on the same few words, and an update takes microseconds
        __nanosleep(spins < 4u ? (250u << spins) : 4000u);
        if (spins > kSpinLimit || ((spins & 63u) == 63u && wave_failed(a.ctrl, lane))) {
            if (lane == 0) atomicOr(&a.ctrl->error, 2u);
            return false;
        }
    }
}

// `flag`: the value of upd_seq[sa + lane] loaded before the walk (the common case: long up to date).
__device__ __forceinline__ bool wait_slabs(const WaveArgs& a, int lane, unsigned warp_id, int sa, int sb, unsigned q, unsigned flag) {
    const bool ok = lane > sb - sa || flag >= q;
    if (__all_sync(0xffffffffu, ok)) return true;
    return wait_slabs_slow(a, lane, warp_id, sa, sb, q);
}

// An updater warp: run posted update sub-tasks until every slab holds the image after block q1 - 1.
__device__ __noinline__ void updater_loop(const WaveArgs& a, int lane, unsigned warp_id, float4* stage) {
    bool ok = false;
    UPROF_DECL;
    for (unsigned idle = 0;;) {
        if (steal_update(a, lane, warp_id, stage)) {
            idle = 0;
            UPROF(3);
            continue;
        }
        UPROF(4);
        if ((idle & 3u) == 0u && slabs_reached(a, lane, 0, a.n_slabs - 1, (unsigned)a.q1, ok)) return;
        __nanosleep(idle < 3u ? (250u << idle) : 2000u);
        if (++idle > kSpinLimit || ((idle & 63u) == 63u && wave_failed(a.ctrl, lane))) {
            if (lane == 0) atomicOr(&a.ctrl->error, 2u);
            return;
        }
    }
}

template <bool SPLINE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) k_wave(const __grid_constant__ WaveArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Geom g = a.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned warp_id = blockIdx.x * kWarpsPerCta + warp;
    const SmemLayout lay = smem_layout(g.kmax);
    float4* s_tab = reinterpret_cast<float4*>(smem_raw);
    PathState* s_state = reinterpret_cast<PathState*>(smem_raw + lay.state_off) + warp * kBatch;
    float2* row = reinterpret_cast<float2*>(smem_raw + lay.row_off) + warp * lay.row_slots;
    stage_table(s_tab, a.tab, g.kmax);
    WaveCtrl* ctrl = a.ctrl;
    const bool planned = a.plan != nullptr;
    if (warp >= kWalkers) {  // updater warps (no CTA-wide barrier follows)
        if (planned)
            updater_loop(a, lane, warp_id, reinterpret_cast<float4*>(smem_raw + wave_stage_off(g.kmax)) + (warp - kWalkers) * (kStageBytes / 16));
        return;
    }
    const long long B = planned ? a.block_size : a.count;
    const long long ipb = (B + a.item - 1) / a.item;  // items per block
    const unsigned long long n_items = planned ? (unsigned long long)(a.q1 - a.q0) * ipb : (unsigned long long)ipb;
    unsigned long long rows = 0, nnz_total = 0, segs = 0;
    const EmitPtrs no_emit{nullptr, nullptr, nullptr, nullptr};
    bool give_up = false;
    PROF_DECL;

    while (!give_up) {
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
            PCT_BOUND(3, first + r >= 0 && first + r < a.n + (planned ? 0 : a.first));
            const Hist hh = load_history(a.H, first + r);
            setup_history(g, hh, s_state[lane]);
        }
        __syncwarp();
        PROF(0);
        for (int p = 0; p < cnt && !give_up; ++p) {
            const PathState& S = s_state[p];
            const int K = S.K;
            if (K < 0) continue;  // skipped history: empty row (R7)
            const int sa = __shfl_sync(0xffffffffu, my_sa, p), sb = __shfl_sync(0xffffffffu, my_sb, p);
            // Issued before the walk, used after it (no latency in the warp's way): the flags of the history's slabs.
            // Relaxed loads: the gather below is issued only
            // after a flag value >= q has arrived, and it reads the L2, where the updater's stores were visible
            // before its release of the flag.
            unsigned flag = 0xffffffffu;
            if (planned && lane <= sb - sa) flag = ld_relaxed_u32(&ctrl->upd_seq[sa + lane]);
            float nrm;
            int nnz;
            walk_history<false, SPLINE>(g, S, s_tab, lane, row, nrm, nnz, no_emit);
            PROF(1);
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
            PROF(2);
            bool bad = false;
            float dot = gather_row_cg(row, lane, C, a.x, lo, span, bad);
            dot = warp_sum(dot);
            nrm = warp_sum(nrm);
            PROF(3);
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
            PROF(4);
        }
        if (planned) {
            // the item has scattered: every lane's reductions are ordered before the counters move
            fence_acq_rel();
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
        PROF(6);
    }
    if (planned && !give_up) {
        // no work left to draw: run update sub-tasks until every slab holds the image after block q1 - 1
        wait_slabs(a, lane, warp_id, 0, a.n_slabs - 1, (unsigned)a.q1, 0u);
    }
    PROF(7);
    PROF_FLUSH;
    nnz_total = (unsigned long long)__reduce_add_sync(0xffffffffu, (unsigned)nnz_total);
    if (lane == 0) {
        atomicAdd(&ctrl->cur[0], rows);
        atomicAdd(&ctrl->cur[1], nnz_total);
        atomicAdd(&ctrl->cur[2], segs);
    }
}

void wave_prof_dump(const char* tag) {
#ifdef PCT_CHECK_BOUNDS
    bounds_dump_tu("wavefront engine");
#endif
#ifdef PCT_WAVE_PROF
    unsigned long long h[16] = {0};
    cudaMemcpyFromSymbol(h, g_wave_prof, sizeof(h));
    double tot = 0;
    for (int i = 0; i < 8; ++i) tot += (double)h[i];
    static const char* names[8] = {"ticket+setup", "walk", "wait", "gather", "scatter", "updates", "signal", "drain"};
    fprintf(stderr, "[wave prof %s]", tag);
    for (int i = 0; i < 8; ++i) fprintf(stderr, " %s %.1f%%", names[i], tot > 0 ? 100.0 * (double)h[i] / tot : 0.0);
    fprintf(stderr, " (total %.3g warp-cycles)\n", tot);
    fprintf(stderr, "[wave prof updaters] sub-tasks %llu, cycles per sub-task: body %.0f, fence %.0f; loop busy %.3g, idle %.3g warp-cycles\n", h[13],
            h[13] ? (double)h[9] / h[13] : 0.0, h[13] ? (double)h[10] / h[13] : 0.0, (double)h[11], (double)h[12]);
    memset(h, 0, sizeof(h));
    cudaMemcpyToSymbol(g_wave_prof, h, sizeof(h));
#else
    (void)tag;
#endif
}

int wave_walkers_per_cta() { return kWalkers; }
size_t wave_smem_need(int nmin) { return wave_smem_bytes(nmin); }

WaveShape wave_shape(const Geom& g) {
    WaveShape s;
    // slabs of at least 4 mm (a typical path spans a millimetre or two in depth) and at most kMaxSlabs of them
    int by_count = (g.nz + kMaxSlabs - 1) / kMaxSlabs;
    int by_mm = (int)(4.0f / g.h + 0.999f);
    s.slab_slices = by_count > by_mm ? by_count : by_mm;
    if (s.slab_slices < 1) s.slab_slices = 1;
    if (s.slab_slices > g.nz) s.slab_slices = g.nz;
    s.n_slabs = (g.nz + s.slab_slices - 1) / s.slab_slices;
    // sub-tasks of about kStageGroups groups of four voxels: one staged chunk of an updater warp
    const long long groups = (long long)s.slab_slices * g.slice_p / 4;
    long long ns = (groups + kStageGroups - 1) / kStageGroups;
    s.n_sub = ns < 1 ? 1 : (ns > 256 ? 256 : (int)ns);
    return s;
}

cudaError_t wave_configure(int nmin, int* grid_out) {
    if (((nmin + 32) >> 5) > 64) return cudaErrorInvalidValue;
    const size_t smem = wave_smem_bytes(nmin);
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
    const long long need = (items + kWalkers - 1) / kWalkers;
    if (need < grid) grid = need < 1 ? 1 : (int)need;
    const size_t smem = wave_smem_bytes(a.g.kmax);
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
