// pct_api.cu -- the C ABI of include/pct.h: argument checks, device memory, the block loop.
// No arithmetic of the path happens here except the host-side fp64 tables of step T / step G
// of the rule, computed once per context.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <stddef.h>

#include <new>
#include <vector>

#include "../../include/pct.h"
#include "pct_internal.h"

using namespace pct;

struct pct_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    Geom g{};
    long long n_voxels = 0;  // nx*ny*nz: the caller's image
    long long n_slots = 0;   // voxels as stored (slices of nxp x nyp, voxel_slot): what the kernels work on
    float* io_buf = nullptr; // n_voxels floats: the image in the caller's order on its way in or out
    float* x = nullptr;
    float2* acc = nullptr;
    float4* tab = nullptr;
    Ctrl* ctrl = nullptr;
    int drop_grid = 0;
    // histories
    bool have_hist = false;
    long long n = 0;
    HistPtrs H{};
    float* tables = nullptr;  // owned: pcos | psin
    void* owned_hist = nullptr;  // owned device block of the host entry point
    // pipelined upload of the host entry point: chunks of 2^20 .. 2^24 histories go up on a copy
    // stream of their own, one event per chunk; the compute stream waits for a chunk only when a
    // DROP block (or an inspection call) first needs it, so the first sweep overlaps the upload
    cudaStream_t copy_stream = nullptr;
    std::vector<cudaEvent_t> chunk_ev;
    std::vector<long long> chunk_end;  // chunk i holds histories [chunk_end[i-1], chunk_end[i])
    size_t chunks_waited = 0;  // events [0, chunks_waited) are already ordered before c->stream's tail
    long long owned_n = 0;     // histories the owned block was sized for (reused by the next upload of the same size)
    int owned_n_proj = 0;
    // processing order of the histories inside each DROP block (k_order_blocks), built per block size
    uint32_t* order = nullptr;
    double l2_bytes = 0.0;      // cudaDevAttrL2CacheSize
    int order_slabs = 4;
    int order_strings = 0;      // 0: built for pct_iterate's blocks, P: for the blocks of P CARP strings
    long long order_block = 0;  // block size the order was built for
    long long order_built = 0;  // blocks [0, order_built) are ordered
    const void* graph_order = nullptr;
    // CARP (pct_iterate_carp): one image, accumulator, control block and stream per string
    int carp_p = 0;
    float* carp_x = nullptr;
    float2* carp_acc = nullptr;
    Ctrl* carp_ctrl = nullptr;
    std::vector<cudaStream_t> carp_stream;
    std::vector<cudaEvent_t> carp_done;
    cudaEvent_t carp_fork = nullptr;
    std::vector<cudaGraphExec_t> carp_graph;  // per string: kGraphPairs (accumulate, update) pairs, like `graph`
    float carp_graph_lambda = 0.f;
    long long carp_graph_block = 0, carp_graph_n = 0;
    const void *carp_graph_hist_key = nullptr, *carp_graph_order = nullptr, *carp_graph_scratch = nullptr;
    int sm_count = 148;
    int opt_order = 1;  // pct_set_option(PCT_OPT_ORDER): depth-slab order of the histories inside a block -- 0 never, 1 by footprint, 2 always
    bool opt_rows_pair = false;
    long long carp_stride = 0;     // voxels between the images / accumulators of two strings (a multiple of four)
    // exact-traversal walk (pct_set_walk): scratch of the lanes' runs, nullptr in the default (midpoint) mode
    float2* exact_scratch = nullptr;
    int exact_cap = 0;
    // total-variation superiorization (pct_set_tvs): off unless tvs_beta0 > 0
    float tvs_beta0 = 0.f, tvs_gamma = 1.f;
    int tvs_levels = 0, tvs_parity = 0;
    float* tvs_grad = nullptr;   // n_slots floats
    TvState* tvs_state = nullptr;
    // cached CUDA graph of kGraphPairs (accumulate, update) pairs
    cudaGraphExec_t graph = nullptr;
    float graph_lambda = 0.f;
    long long graph_block = 0, graph_n = 0;
    const void* graph_hist_key = nullptr;
    long long last_n_iter_hist = 0;
    char err[512] = {0};
};

static thread_local char g_create_err[512] = {0};
static int tvs_step(pct_ctx* c, float* x, cudaStream_t s);
static int exact_scratch_alloc(pct_ctx* c);
static const int kGraphPairs = 64;
// Upload chunks (histories): the first one is small so that the first DROP blocks start after about a
// millisecond, the following ones double up to 2^24 (64 MB per float field) so that a 19 GB upload is
// a few hundred copy calls -- more would overflow the copy stream's submission queue and block the
// host inside pct_set_histories_host while the compute stream sits idle.
static const long long kUploadChunkMin = 1LL << 20, kUploadChunkMax = 1LL << 24;

static int fail(pct_ctx* c, int code, const char* fmt, const char* detail = "") {
    char* dst = c ? c->err : g_create_err;
    snprintf(dst, 512, fmt, detail);
    return code;
}
// Every entry point runs on the context's device, whatever device the calling thread has current, and restores it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};
#define CUDA_TRY(c, call)                                                                  \
    do {                                                                                   \
        cudaError_t e__ = (call);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            (void)cudaGetLastError();                                                      \
            return fail((c), e__ == cudaErrorMemoryAllocation ? PCT_ENOMEM : PCT_ECUDA,    \
                        #call ": %s", cudaGetErrorString(e__));                            \
        }                                                                                  \
    } while (0)

// Rule step T: Sigma1^-1 at depth s = k*h, fp64 closed forms, rounded once to fp32.
//   a_j = A_CM[j] * 0.1^j (j successive multiplications by 0.1) * 8192
//   C = sum a_j s^(j+1)/(j+1), B = sum a_j s^(j+2)/((j+1)(j+2)), A = sum 2 a_j s^(j+3)/((j+1)(j+2)(j+3))
//   W = (1 + 0.038 ln(s/361))^2 (A C - B^2);  (p11, p12, p22) = (C/W, -B/W, A/W)
static void sigma1_inverse_table(float h32, int kmax, float4* out) {
    static const double A_CM[6] = {7.457e-6, 4.548e-7, -5.777e-8, 1.301e-8, -9.228e-10, 2.687e-11};
    double a[6];
    for (int j = 0; j < 6; ++j) {
        double v = A_CM[j];
        for (int i = 0; i < j; ++i) v *= 0.1;
        a[j] = v * 8192.0;
    }
    const double h = (double)h32;
    out[0] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int k = 1; k <= kmax; ++k) {
        const double s = (double)k * h;
        double A = 0.0, B = 0.0, C = 0.0, sp = s;
        for (int j = 0; j < 6; ++j) {
            C += a[j] * sp / (double)(j + 1);
            B += a[j] * sp * s / (double)((j + 1) * (j + 2));
            A += 2.0 * a[j] * sp * s * s / (double)((j + 1) * (j + 2) * (j + 3));
            sp *= s;
        }
        const double gl = 1.0 + 0.038 * log(s / 361.0);
        const double W = gl * gl * (A * C - B * B);
        // .w = s1 = float(k) * h, the ONE fp32 product of rule step 3b (identical to __fmul_rn(__int2float_rn(k), h)
        // on the device: an exact int -> float conversion and one correctly rounded multiplication)
        const volatile float s1 = (float)k * h32;
        out[k] = make_float4((float)(C / W), (float)(-B / W), (float)(A / W), s1);
    }
}

static void drop_graph(pct_ctx* c) {
    if (c->graph) {
        cudaGraphExecDestroy(c->graph);
        c->graph = nullptr;
    }
    for (cudaGraphExec_t g : c->carp_graph)
        if (g) cudaGraphExecDestroy(g);
    c->carp_graph.clear();
}

// Make the compute stream wait for the upload of histories [0, upto) (all of them: upto < 0).
static int wait_upload(pct_ctx* c, long long upto) {
    const size_t all = c->chunk_ev.size();
    while (c->chunks_waited < all && (upto < 0 || c->chunks_waited == 0 || c->chunk_end[c->chunks_waited - 1] < upto)) {
        CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->chunk_ev[c->chunks_waited], 0));
        ++c->chunks_waited;
    }
    return PCT_OK;
}

// The order buffer for this block size (4 B per history); without memory for it the blocks run in the
// caller's order.  Slabs: image + accumulator (12 B per voxel) of one slab take a quarter of the L2, at
// least 4 (measured at 256 x 256 x 160, 126 MB: 440 -> 317 us per 2e5-history block with 4 slabs, 318
// with 8, 323 with 16; at 256 x 256 x 128, 101 MB: 169.3 -> 166.9 us, k_update 23.2 -> 24.3 us).
// (strings = 0: the DROP blocks of pct_iterate; strings = P: the blocks of the P CARP strings, which count
// from each string's first history and work on P images at once)
static void prepare_order(pct_ctx* c, long long block_size, int strings = 0) {
    const double images = strings > 0 ? (double)strings : 1.0;
    const double l2 = c->l2_bytes > 0.0 ? c->l2_bytes : 128.0e6;
    // ordering pays when image + accumulator do not fit the L2; for a grid that fits it is a wash (256 x 256 x
    // 128, 101 MB: sweep 906 -> 910 ms, and every upload would pay the sort), so such grids keep the caller's
    // order and its coalesced history loads
    const int mode = c->opt_order;  // pct_set_option(PCT_OPT_ORDER): 0 never, 1 by footprint (default), 2 always
    const bool wanted = mode == 2 || (mode == 1 && 12.0 * images * (double)c->n_slots > 0.85 * l2);
    if (!wanted || block_size < 1024) {  // (small blocks: nothing to gain)
        if (c->order) cudaFree(c->order);
        c->order = nullptr;
        c->order_block = 0;
        return;
    }
    const double per_slab = 0.25 * l2;
    const double want = ceil(12.0 * images * (double)c->n_slots / per_slab);
    c->order_slabs = want < 4.0 ? 4 : (want > 64.0 ? 64 : (int)want);
    if (c->order && c->order_block == block_size && c->order_strings == strings) return;
    if (!c->order && cudaMalloc(&c->order, sizeof(uint32_t) * (size_t)c->n) != cudaSuccess) {
        (void)cudaGetLastError();
        c->order = nullptr;
    }
    c->order_block = block_size;
    c->order_strings = strings;
    c->order_built = 0;
}

// Order DROP blocks [order_built, upto) (their histories must be on the device or on their way in c->stream's order).
static int build_order(pct_ctx* c, long long block_size, long long upto) {
    if (!c->order || upto <= c->order_built) return PCT_OK;
    CUDA_TRY(c, launch_order_blocks(c->H, c->g, c->n, block_size, c->order_built, upto - c->order_built, c->order_slabs, c->order, c->stream));
    c->order_built = upto;
    return PCT_OK;
}

static void release_histories(pct_ctx* c) {
    drop_graph(c);
    if (c->order) cudaFree(c->order);
    c->order = nullptr;
    c->order_block = 0;
    c->order_built = 0;
    if (!c->chunk_ev.empty()) {
        if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
        for (cudaEvent_t e : c->chunk_ev) cudaEventDestroy(e);
        c->chunk_ev.clear();
    }
    c->chunk_end.clear();
    c->chunks_waited = 0;
    if (c->owned_hist) cudaFree(c->owned_hist);
    if (c->tables) cudaFree(c->tables);
    c->owned_hist = nullptr;
    c->owned_n = 0;
    c->tables = nullptr;
    c->have_hist = false;
    c->n = 0;
}

extern "C" const char* pct_version(void) { return "pct-b200 0.1 sm_100a"; }

extern "C" const char* pct_last_error(const pct_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

extern "C" int pct_create(pct_ctx** out, int nx, int ny, int nz, float h, float u_in, float u_out, void* stream) {
    if (!out) return fail(nullptr, PCT_EINVAL, "pct_create: out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(nullptr, PCT_EINVAL, "pct_create: grid dimensions must be >= 1");
    if ((long long)nx * ny * nz >= (1LL << 31)) return fail(nullptr, PCT_EINVAL, "pct_create: nx*ny*nz must be < 2^31");
    if (!(h > 0.0f) || !isfinite(h)) return fail(nullptr, PCT_EINVAL, "pct_create: voxel_mm must be positive and finite");
    const int nmin = nx < ny ? nx : ny;
    if (((nmin + 32) >> 5) > 64 || drop_smem_bytes(nmin) + 1024 > (size_t)227 * 1024) {  // (1 KB: the kernels' static shared memory)
        snprintf(g_create_err, 512, "pct_create: min(nx,ny) = %d is too wide: the rows of a CTA's warps and the staged tables need %zu B of "
                 "shared memory, a B200 offers %d less 1 KB for the kernels' own (min(nx,ny) <= 1318)", nmin, drop_smem_bytes(nmin), 227 * 1024);
        return PCT_EINVAL;
    }
    // rule step G (fp32, this operation order)
    Geom g{};
    g.nx = nx; g.ny = ny; g.nz = nz; g.nmin = nmin;
    g.h = h;
    g.inv_h = 1.0f / h;
    const float R = (0.5f * h) * (float)nmin;
    g.R = R;
    g.R2 = R * R;
    g.zmax = (0.5f * (float)nz) * h;
    g.u_in = u_in; g.u_out = u_out;
    g.hx = 0.5f * (float)nx; g.hy = 0.5f * (float)ny; g.hz = 0.5f * (float)nz;
    g.fnx = (float)nx; g.fny = (float)ny; g.fnz = (float)nz;
    g.inv_step = g.inv_h;  // (pct_set_step: one voxel edge per node by default, R9)
    g.kmax = nmin;
    if (!(u_in <= -R) || !(u_out >= R) || !isfinite(u_in) || !isfinite(u_out))
        return fail(nullptr, PCT_EINVAL, "pct_create: tracker planes must lie outside the hull (u_in <= -R_h, u_out >= R_h)");
    pct_ctx* c = new (std::nothrow) pct_ctx;
    if (!c) return fail(nullptr, PCT_ENOMEM, "pct_create: out of host memory");
    c->g = g;
    c->n_voxels = (long long)nx * ny * nz;
    c->g.nxp = (nx + 1) & ~1;
    c->g.slice_p = c->g.nxp * ((ny + 1) & ~1);
    c->n_slots = (long long)c->g.slice_p * nz;
    if (c->n_slots >= (1LL << 31)) {
        delete c;
        return fail(nullptr, PCT_EINVAL, "pct_create: the stored image (nx, ny rounded up to even) must have < 2^31 voxels");
    }
    c->stream = (cudaStream_t)stream;
    int rc = PCT_OK;
    auto body = [&]() -> int {
        CUDA_TRY(nullptr, cudaGetDevice(&c->device));
        int l2 = 0;
        CUDA_TRY(nullptr, cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, c->device));
        c->l2_bytes = (double)l2;
        CUDA_TRY(nullptr, cudaMalloc(&c->x, sizeof(float) * c->n_slots));
        CUDA_TRY(nullptr, cudaMalloc(&c->acc, sizeof(float2) * c->n_slots));
        CUDA_TRY(nullptr, cudaMalloc(&c->io_buf, sizeof(float) * c->n_voxels));
        CUDA_TRY(nullptr, cudaMalloc(&c->tab, sizeof(float4) * (2 * nmin + 1)));  // (room for the half-voxel step)
        CUDA_TRY(nullptr, cudaMalloc(&c->ctrl, sizeof(Ctrl)));
        CUDA_TRY(nullptr, cudaMemsetAsync(c->x, 0, sizeof(float) * c->n_slots, c->stream));
        CUDA_TRY(nullptr, cudaMemsetAsync(c->acc, 0, sizeof(float2) * c->n_slots, c->stream));
        CUDA_TRY(nullptr, cudaMemsetAsync(c->ctrl, 0, sizeof(Ctrl), c->stream));
        float4* tab = (float4*)malloc(sizeof(float4) * (nmin + 1));
        if (!tab) return fail(nullptr, PCT_ENOMEM, "pct_create: out of host memory");
        sigma1_inverse_table(h, nmin, tab);
        cudaError_t e = cudaMemcpyAsync(c->tab, tab, sizeof(float4) * (nmin + 1), cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        free(tab);
        CUDA_TRY(nullptr, e);
        CUDA_TRY(nullptr, cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));
        // the per-warp row buffer and the two staged copies of the table must fit the shared memory of an SM
        int smem_max = 0;
        CUDA_TRY(nullptr, cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
        if (drop_smem_bytes(nmin) + 1024 > (size_t)smem_max) {
            snprintf(g_create_err, 512, "pct_create: min(nx,ny) = %d needs %zu B of shared memory per CTA, the device offers %d",
                     nmin, drop_smem_bytes(nmin), smem_max);
            return PCT_EINVAL;
        }
        CUDA_TRY(nullptr, drop_configure(nmin, &c->drop_grid));
        return PCT_OK;
    };
    rc = body();
    if (rc != PCT_OK) {
        char keep[512];
        memcpy(keep, g_create_err, 512);
        pct_destroy(c);
        memcpy(g_create_err, keep, 512);
        return rc;
    }
    *out = c;
    return PCT_OK;
}

static void release_carp(pct_ctx* c) {
    for (cudaGraphExec_t g : c->carp_graph)  // (they hold the strings' buffers)
        if (g) cudaGraphExecDestroy(g);
    c->carp_graph.clear();
    for (cudaStream_t s : c->carp_stream) {
        cudaStreamSynchronize(s);
        cudaStreamDestroy(s);
    }
    for (cudaEvent_t e : c->carp_done) cudaEventDestroy(e);
    c->carp_stream.clear();
    c->carp_done.clear();
    if (c->carp_fork) cudaEventDestroy(c->carp_fork);
    c->carp_fork = nullptr;
    if (c->carp_x) cudaFree(c->carp_x);
    if (c->carp_acc) cudaFree(c->carp_acc);
    if (c->carp_ctrl) cudaFree(c->carp_ctrl);
    c->carp_x = nullptr;
    c->carp_acc = nullptr;
    c->carp_ctrl = nullptr;
    c->carp_p = 0;
}

extern "C" void pct_destroy(pct_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    release_carp(c);
    release_histories(c);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->x) cudaFree(c->x);
    if (c->io_buf) cudaFree(c->io_buf);
    if (c->acc) cudaFree(c->acc);
    if (c->tab) cudaFree(c->tab);
    if (c->ctrl) cudaFree(c->ctrl);
    if (c->exact_scratch) cudaFree(c->exact_scratch);
    if (c->tvs_grad) cudaFree(c->tvs_grad);
    if (c->tvs_state) cudaFree(c->tvs_state);
    (void)cudaGetLastError();
    delete c;
}

static bool is_device_ptr(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static int check_histories(pct_ctx* c, long long n, const pct_histories* h, bool want_device) {
    if (!c) return PCT_EINVAL;
    if (!h) return fail(c, PCT_EINVAL, "pct_set_histories: h is NULL");
    if (n < 1 || n >= (1LL << 40)) return fail(c, PCT_EINVAL, "pct_set_histories: n must be in [1, 2^40)");
    if (h->n_proj < 1 || h->n_proj > 65536) return fail(c, PCT_EINVAL, "pct_set_histories: n_proj must be in [1, 65536]");
    const void* ptrs[12] = {h->entry_t, h->entry_v, h->exit_t, h->exit_v, h->entry_dt, h->entry_dv,
                            h->exit_dt, h->exit_dv, h->wepl, h->proj, h->proj_cos, h->proj_sin};
    for (int i = 0; i < 12; ++i) {
        if (!ptrs[i]) return fail(c, PCT_EINVAL, "pct_set_histories: null array pointer");
        if (is_device_ptr(ptrs[i]) != want_device)
            return fail(c, PCT_EINVAL, want_device ? "pct_set_histories: arrays must be device memory"
                                                   : "pct_set_histories_host: arrays must be host memory");
    }
    return PCT_OK;
}

extern "C" int pct_set_histories(pct_ctx* c, int64_t n, const pct_histories* h) {
    int rc = check_histories(c, n, h, true);
    if (rc) return rc;
    DeviceGuard guard(c->device);
    release_histories(c);
    CUDA_TRY(c, cudaMalloc(&c->tables, sizeof(float) * 2 * h->n_proj));
    CUDA_TRY(c, cudaMemcpyAsync(c->tables, h->proj_cos, sizeof(float) * h->n_proj, cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->tables + h->n_proj, h->proj_sin, sizeof(float) * h->n_proj, cudaMemcpyDeviceToDevice, c->stream));
    c->H = HistPtrs{h->entry_t, h->entry_v, h->exit_t, h->exit_v, h->entry_dt, h->entry_dv, h->exit_dt, h->exit_dv,
                    h->wepl, h->proj, c->tables, c->tables + h->n_proj, h->n_proj};
    c->n = n;
    c->have_hist = true;
    return PCT_OK;
}

extern "C" int pct_set_histories_xyz(pct_ctx* c, int64_t n, const pct_histories_xyz* h) {
    if (!c) return PCT_EINVAL;
    if (!h) return fail(c, PCT_EINVAL, "pct_set_histories_xyz: h is NULL");
    if (n < 1 || n >= (1LL << 40)) return fail(c, PCT_EINVAL, "pct_set_histories_xyz: n must be in [1, 2^40)");
    if (h->n_proj < 1 || h->n_proj > 65536) return fail(c, PCT_EINVAL, "pct_set_histories_xyz: n_proj must be in [1, 65536]");
    const void* ptrs[14] = {h->entry_x, h->entry_y, h->entry_z, h->exit_x, h->exit_y, h->exit_z, h->entry_dt, h->entry_dv,
                            h->exit_dt, h->exit_dv, h->wepl, h->proj, h->proj_cos, h->proj_sin};
    for (int i = 0; i < 14; ++i)
        if (!ptrs[i] || !is_device_ptr(ptrs[i])) return fail(c, PCT_EINVAL, "pct_set_histories_xyz: arrays must be device memory");
    DeviceGuard guard(c->device);
    release_histories(c);
    // four owned arrays (positions at the tracker planes, each padded to 256 B); slopes, WEPL and proj stay borrowed
    const size_t fa = ((sizeof(float) * (size_t)n + 255) / 256) * 256;
    cudaError_t e = cudaMalloc(&c->owned_hist, 4 * fa);
    if (e == cudaSuccess) e = cudaMalloc(&c->tables, sizeof(float) * 2 * h->n_proj);
    if (e != cudaSuccess) {
        release_histories(c);
        CUDA_TRY(c, e);
    }
    c->owned_n = -1;  // (not a block of the host entry point: never reused by it)
    float* d[4];
    for (int i = 0; i < 4; ++i) d[i] = (float*)((char*)c->owned_hist + i * fa);
    float* pc = c->tables;
    float* ps = c->tables + h->n_proj;
    int rc = PCT_OK;
    auto body = [&]() -> int {
        CUDA_TRY(c, cudaMemcpyAsync(pc, h->proj_cos, sizeof(float) * h->n_proj, cudaMemcpyDeviceToDevice, c->stream));
        CUDA_TRY(c, cudaMemcpyAsync(ps, h->proj_sin, sizeof(float) * h->n_proj, cudaMemcpyDeviceToDevice, c->stream));
        CUDA_TRY(c, launch_xyz_to_beam(c->g.u_in, n, h->entry_x, h->entry_y, h->entry_z, h->entry_dt, h->entry_dv, h->proj, pc, ps, h->n_proj,
                                       d[0], d[1], c->stream));
        CUDA_TRY(c, launch_xyz_to_beam(c->g.u_out, n, h->exit_x, h->exit_y, h->exit_z, h->exit_dt, h->exit_dv, h->proj, pc, ps, h->n_proj,
                                       d[2], d[3], c->stream));
        return PCT_OK;
    };
    rc = body();
    if (rc != PCT_OK) {
        char keep[512];
        memcpy(keep, c->err, 512);
        release_histories(c);
        memcpy(c->err, keep, 512);
        return rc;
    }
    c->H = HistPtrs{d[0], d[1], d[2], d[3], h->entry_dt, h->entry_dv, h->exit_dt, h->exit_dv, h->wepl, h->proj, pc, ps, h->n_proj};
    c->n = n;
    c->have_hist = true;
    return PCT_OK;
}

static int set_histories_host_impl(pct_ctx* c, int64_t n, const pct_histories* h);

extern "C" int pct_set_histories_host(pct_ctx* c, int64_t n, const pct_histories* h) {
    int rc = check_histories(c, n, h, false);
    if (rc) return rc;
    DeviceGuard guard(c->device);
    rc = set_histories_host_impl(c, n, h);
    if (rc != PCT_OK) {  // a failure part-way (allocation, a copy that could not be enqueued) leaves NO histories set
        char keep[512];
        memcpy(keep, c->err, 512);
        if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
        release_histories(c);
        (void)cudaGetLastError();
        memcpy(c->err, keep, 512);
    }
    return rc;
}

static int set_histories_host_impl(pct_ctx* c, int64_t n, const pct_histories* h) {
    // one owned block: 9 float arrays (each padded to 256 B) + the uint16 array
    const size_t fa = ((sizeof(float) * (size_t)n + 255) / 256) * 256;
    const size_t total = 9 * fa + ((sizeof(uint16_t) * (size_t)n + 255) / 256) * 256;
    if (c->owned_hist && c->tables && c->owned_n == n && c->owned_n_proj == h->n_proj) {
        // a new set of the same size (the next acquisition through the same pipeline): the device block,
        // the tables and the cached graph are reused -- no 19 GB cudaFree + cudaMalloc per upload.  The
        // new upload is ordered after everything already enqueued that reads the old histories.
        if (c->copy_stream) CUDA_TRY(c, cudaStreamSynchronize(c->copy_stream));
        for (cudaEvent_t e : c->chunk_ev) cudaEventDestroy(e);
        c->chunk_ev.clear();
        c->chunk_end.clear();
        c->chunks_waited = 0;
        c->order_built = 0;  // same buffer, new histories: the blocks are ordered again as they arrive
        cudaEvent_t tail = nullptr;
        CUDA_TRY(c, cudaEventCreateWithFlags(&tail, cudaEventDisableTiming));
        cudaError_t e = cudaEventRecord(tail, c->stream);
        if (!c->copy_stream && e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, tail, 0);
        cudaEventDestroy(tail);
        CUDA_TRY(c, e);
    } else {
        release_histories(c);
        CUDA_TRY(c, cudaMalloc(&c->owned_hist, total));
        CUDA_TRY(c, cudaMalloc(&c->tables, sizeof(float) * 2 * h->n_proj));
        c->owned_n = n;
        c->owned_n_proj = h->n_proj;
    }
    const float* src[9] = {h->entry_t, h->entry_v, h->exit_t, h->exit_v, h->entry_dt, h->entry_dv, h->exit_dt, h->exit_dv, h->wepl};
    float* dst[9];
    for (int i = 0; i < 9; ++i) dst[i] = (float*)((char*)c->owned_hist + i * fa);
    uint16_t* dproj = (uint16_t*)((char*)c->owned_hist + 9 * fa);
    if (!c->copy_stream) CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    // chunk by chunk, all ten fields of a chunk together, one event per chunk (the tables ride with chunk 0)
    CUDA_TRY(c, cudaMemcpyAsync(c->tables, h->proj_cos, sizeof(float) * h->n_proj, cudaMemcpyHostToDevice, c->copy_stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->tables + h->n_proj, h->proj_sin, sizeof(float) * h->n_proj, cudaMemcpyHostToDevice, c->copy_stream));
    long long chunk = kUploadChunkMin;
    for (long long i0 = 0; i0 < n; i0 += chunk, chunk = chunk < kUploadChunkMax && i0 >= 2 * kUploadChunkMin ? 2 * chunk : chunk) {
        const size_t cnt = (size_t)(n - i0 < chunk ? n - i0 : chunk);
        for (int i = 0; i < 9; ++i)
            CUDA_TRY(c, cudaMemcpyAsync(dst[i] + i0, src[i] + i0, sizeof(float) * cnt, cudaMemcpyHostToDevice, c->copy_stream));
        CUDA_TRY(c, cudaMemcpyAsync(dproj + i0, h->proj + i0, sizeof(uint16_t) * cnt, cudaMemcpyHostToDevice, c->copy_stream));
        cudaEvent_t ev = nullptr;
        CUDA_TRY(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        c->chunk_ev.push_back(ev);
        c->chunk_end.push_back(i0 + (long long)cnt);
        CUDA_TRY(c, cudaEventRecord(ev, c->copy_stream));
    }
    c->H = HistPtrs{dst[0], dst[1], dst[2], dst[3], dst[4], dst[5], dst[6], dst[7], dst[8], dproj,
                    c->tables, c->tables + h->n_proj, h->n_proj};
    c->n = n;
    c->have_hist = true;
    return PCT_OK;
}

static DropArgs drop_args(pct_ctx* c, long long block_size, long long first, long long count) {
    DropArgs a{};
    a.g = c->g;
    a.H = c->H;
    a.n = c->n;
    a.block_size = block_size;
    a.first = first;
    a.count = count;
    a.x = c->x;
    a.acc = c->acc;
    a.tab = c->tab;
    a.ctrl = c->ctrl;
    a.order = first < 0 ? c->order : nullptr;
    a.scratch = c->exact_scratch;
    a.cap_lane = c->exact_cap;
    return a;
}

// One DROP block: accumulate over the block a.ctrl->block points at, then update a.x and advance the block index.
static int enqueue_pair(pct_ctx* c, const DropArgs& a, int grid, float lambda, long long n_blocks, cudaStream_t s) {
    CUDA_TRY(c, launch_drop_block(a, grid, s));
    CUDA_TRY(c, launch_update(const_cast<float*>(a.x), a.acc, c->n_slots, lambda, a.ctrl, n_blocks, c->order != nullptr, s));
    return PCT_OK;
}

// kGraphPairs such pairs as one executable graph (the block index lives on the device, so one graph serves every block).
static int capture_pairs(pct_ctx* c, const DropArgs& a, int grid, float lambda, long long n_blocks, cudaGraphExec_t* out) {
    cudaStream_t cap = nullptr;
    CUDA_TRY(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaGraph_t gr = nullptr;
    int rc = PCT_OK;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        for (int i = 0; i < kGraphPairs && rc == PCT_OK; ++i) rc = enqueue_pair(c, a, grid, lambda, n_blocks, cap);
        e = cudaStreamEndCapture(cap, &gr);
    }
    if (e == cudaSuccess && rc == PCT_OK) e = cudaGraphInstantiate(out, gr, 0);
    if (gr) cudaGraphDestroy(gr);
    cudaStreamDestroy(cap);
    if (rc != PCT_OK) return rc;
    CUDA_TRY(c, e);
    return PCT_OK;
}


extern "C" int pct_iterate(pct_ctx* c, float lambda, int64_t block_size, int n_iter) {
    if (!c) return PCT_EINVAL;
    if (!c->have_hist) return fail(c, PCT_ESTATE, "pct_iterate: no histories set");
    if (!(lambda > 0.0f) || !(lambda < 2.0f)) return fail(c, PCT_EINVAL, "pct_iterate: lambda must be in (0, 2)");
    if (block_size < 1 || block_size > (1LL << 24)) return fail(c, PCT_EINVAL, "pct_iterate: block_size must be in [1, 2^24]");
    if (n_iter < 0) return fail(c, PCT_EINVAL, "pct_iterate: n_iter must be >= 0");
    if (n_iter == 0) return PCT_OK;
    DeviceGuard guard(c->device);
    const bool tvs = c->tvs_beta0 > 0.0f;  // a step on the image that enters every block: launches go out one by one
    const long long n_blocks = (c->n + block_size - 1) / block_size;
    const long long pairs = n_blocks * (long long)n_iter;
    CUDA_TRY(c, cudaMemsetAsync(c->ctrl, 0, sizeof(Ctrl), c->stream));
    prepare_order(c, block_size);
    if (c->chunks_waited == c->chunk_ev.size()) {  // every history is on the device: order all blocks in one launch
        int rc = build_order(c, block_size, n_blocks);
        if (rc) return rc;
    }
    const DropArgs a = drop_args(c, block_size, -1, 0);
    long long done = 0;
    if (pairs >= 2 * kGraphPairs && !tvs) {
        const bool reuse = c->graph && c->graph_lambda == lambda && c->graph_block == block_size && c->graph_n == c->n &&
                           c->graph_hist_key == (const void*)c->H.t_in && c->graph_order == (const void*)c->order;
        if (!reuse) {
            drop_graph(c);
            if (int rc = capture_pairs(c, a, c->drop_grid, lambda, n_blocks, &c->graph)) return rc;
            c->graph_lambda = lambda;
            c->graph_block = block_size;
            c->graph_n = c->n;
            c->graph_hist_key = (const void*)c->H.t_in;
            c->graph_order = (const void*)c->order;
        }
        for (; done + kGraphPairs <= pairs; done += kGraphPairs) {
            // blocks done .. done+63 of the first sweep need the histories below (done + 64) * block_size
            int rc = wait_upload(c, done + kGraphPairs <= n_blocks ? (done + kGraphPairs) * block_size : -1);
            if (rc == PCT_OK) rc = build_order(c, block_size, done + kGraphPairs <= n_blocks ? done + kGraphPairs : n_blocks);
            if (rc) return rc;
            CUDA_TRY(c, cudaGraphLaunch(c->graph, c->stream));
        }
    }
    for (; done < pairs; ++done) {
        int rc = wait_upload(c, done < n_blocks ? (done + 1) * block_size : -1);
        if (rc == PCT_OK) rc = build_order(c, block_size, done < n_blocks ? done + 1 : n_blocks);
        if (rc == PCT_OK && tvs) rc = tvs_step(c, c->x, c->stream);
        if (rc == PCT_OK) rc = enqueue_pair(c, a, c->drop_grid, lambda, n_blocks, c->stream);
        if (rc) return rc;
    }
    return PCT_OK;
}

// CARP (Fig. 2; R27-R29).  Every string runs its DROP sweep on a stream of its
// own, with its own image copy, accumulator and control block, so the strings' kernels overlap: the tail of
// one string's block launch and its update kernel are filled by the other strings' blocks.
extern "C" int pct_iterate_carp(pct_ctx* c, float lambda, int64_t block_size, int n_iter, int n_strings) {
    if (!c) return PCT_EINVAL;
    if (!c->have_hist) return fail(c, PCT_ESTATE, "pct_iterate_carp: no histories set");
    if (!(lambda > 0.0f) || !(lambda < 2.0f)) return fail(c, PCT_EINVAL, "pct_iterate_carp: lambda must be in (0, 2)");
    if (block_size < 1 || block_size > (1LL << 24)) return fail(c, PCT_EINVAL, "pct_iterate_carp: block_size must be in [1, 2^24]");
    if (n_iter < 0) return fail(c, PCT_EINVAL, "pct_iterate_carp: n_iter must be >= 0");
    if (n_strings < 1 || n_strings > 64 || (long long)n_strings > c->n)
        return fail(c, PCT_EINVAL, "pct_iterate_carp: n_strings must be in [1, min(64, n)]");
    if (n_iter == 0) return PCT_OK;
    if (int rc = wait_upload(c, -1)) return rc;
    const int P = n_strings;
    const long long M = c->n_slots;  // (the strings' images live in storage order like the context's)
    DeviceGuard guard(c->device);
    // every string's image and accumulator start on a 16-byte boundary (the update reads them 128 bits at a time)
    const long long stride = (M + 3) & ~3LL;
    if (c->carp_p != P) {
        release_carp(c);
        c->carp_stride = stride;
        CUDA_TRY(c, cudaMalloc(&c->carp_x, sizeof(float) * (size_t)stride * P));
        CUDA_TRY(c, cudaMalloc(&c->carp_acc, sizeof(float2) * (size_t)stride * P));
        CUDA_TRY(c, cudaMalloc(&c->carp_ctrl, sizeof(Ctrl) * P));
        CUDA_TRY(c, cudaMemsetAsync(c->carp_acc, 0, sizeof(float2) * (size_t)stride * P, c->stream));
        CUDA_TRY(c, cudaEventCreateWithFlags(&c->carp_fork, cudaEventDisableTiming));
        for (int p = 0; p < P; ++p) {
            cudaStream_t s = nullptr;
            cudaEvent_t e = nullptr;
            CUDA_TRY(c, cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
            c->carp_stream.push_back(s);
            CUDA_TRY(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            c->carp_done.push_back(e);
        }
        c->carp_p = P;
    }
    prepare_order(c, block_size, P);
    if (c->order && c->order_built == 0) {  // every string's blocks, ordered by depth slab (k_order_blocks)
        for (int p = 0; p < P; ++p) {
            const long long lo = (long long)(((__int128)p * c->n) / P), hi = (long long)(((__int128)(p + 1) * c->n) / P);
            HistPtrs Hs = c->H;
            Hs.t_in += lo; Hs.v_in += lo; Hs.dt_in += lo; Hs.dv_in += lo;
            CUDA_TRY(c, launch_order_blocks(Hs, c->g, hi - lo, block_size, 0, (hi - lo + block_size - 1) / block_size,
                                            c->order_slabs, c->order + lo, c->stream));
        }
        c->order_built = 1;
    }
    {  // the strings' cached graphs hold these arguments
        const bool same = c->carp_graph_lambda == lambda && c->carp_graph_block == block_size && c->carp_graph_n == c->n &&
                          c->carp_graph_hist_key == (const void*)c->H.t_in && c->carp_graph_order == (const void*)c->order &&
                          c->carp_graph_scratch == (const void*)c->exact_scratch && (int)c->carp_graph.size() == P;
        if (!same) {
            for (cudaGraphExec_t g : c->carp_graph)
                if (g) cudaGraphExecDestroy(g);
            c->carp_graph.assign(P, nullptr);
            c->carp_graph_lambda = lambda;
            c->carp_graph_block = block_size;
            c->carp_graph_n = c->n;
            c->carp_graph_hist_key = (const void*)c->H.t_in;
            c->carp_graph_order = (const void*)c->order;
            c->carp_graph_scratch = (const void*)c->exact_scratch;
        }
    }
    for (int it = 0; it < n_iter; ++it) {
        if (c->tvs_beta0 > 0.0f)  // "In CARP, TVS is applied just once to the initial solution at the start of each iteration"
            if (int rc = tvs_step(c, c->x, c->stream)) return rc;
        CUDA_TRY(c, cudaEventRecord(c->carp_fork, c->stream));  // x (and, the first time, the zeroed accumulators) are ready
        for (int p = 0; p < P; ++p) {
            cudaStream_t s = c->carp_stream[p];
            const long long lo = (long long)(((__int128)p * c->n) / P), hi = (long long)(((__int128)(p + 1) * c->n) / P);
            float* xs = c->carp_x + (size_t)p * stride;
            CUDA_TRY(c, cudaStreamWaitEvent(s, c->carp_fork, 0));
            CUDA_TRY(c, cudaMemcpyAsync(xs, c->x, sizeof(float) * M, cudaMemcpyDeviceToDevice, s));  // the common x0
            CUDA_TRY(c, cudaMemsetAsync(c->carp_ctrl + p, 0, sizeof(Ctrl), s));
            DropArgs a = drop_args(c, block_size, -1, 0);
            a.H.t_in += lo; a.H.v_in += lo; a.H.t_out += lo; a.H.v_out += lo;
            a.H.dt_in += lo; a.H.dv_in += lo; a.H.dt_out += lo; a.H.dv_out += lo;
            a.H.wepl += lo; a.H.proj += lo;
            a.n = hi - lo;
            a.x = xs;
            a.acc = c->carp_acc + (size_t)p * stride;
            if (a.scratch)  // exact-traversal mode: the strings' kernels run concurrently, each on its own part of the scratch
                a.scratch = (float2*)((char*)a.scratch + (size_t)p * exact_scratch_bytes(c->g.kmax, (c->drop_grid + P - 1) / P, nullptr));
            a.ctrl = c->carp_ctrl + p;
            a.order = c->order ? c->order + lo : nullptr;
            const long long n_blocks = (a.n + block_size - 1) / block_size;
            // every string gets its share of the CTA slots: P block launches in flight side by side, each P times
            // longer (measured at 256 x 256 x 128, 1e8 histories: the same rate as whole-grid launches, 5.4e8 /s)
            const int grid = (c->drop_grid + P - 1) / P;
            long long b = 0;
            if (n_blocks >= 2 * kGraphPairs) {  // the string's block loop from a graph of its own, as in pct_iterate
                if ((int)c->carp_graph.size() != P) c->carp_graph.assign(P, nullptr);
                if (!c->carp_graph[p])
                    if (int rc = capture_pairs(c, a, grid, lambda, n_blocks, &c->carp_graph[p])) return rc;
                for (; b + kGraphPairs <= n_blocks; b += kGraphPairs) CUDA_TRY(c, cudaGraphLaunch(c->carp_graph[p], s));
            }
            for (; b < n_blocks; ++b)
                if (int rc = enqueue_pair(c, a, grid, lambda, n_blocks, s)) return rc;
            CUDA_TRY(c, cudaEventRecord(c->carp_done[p], s));
            CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->carp_done[p], 0));
        }
        CUDA_TRY(c, launch_mean(c->x, c->carp_x, P, M, stride, c->stream));
        // pct_get_stats: the counters of the strings' sweeps, added up
        CUDA_TRY(c, launch_sum_stats(c->ctrl->last, c->carp_ctrl[0].last, sizeof(Ctrl), P, c->stream));
    }
    return PCT_OK;
}

// ---- total-variation superiorization (R31) ----------------------------------------------

static int tvs_step(pct_ctx* c, float* x, cudaStream_t s) {
    CUDA_TRY(c, launch_tvs_step(x, c->tvs_grad, c->g, c->n_slots, c->tvs_state, c->tvs_parity, c->tvs_levels, c->tvs_gamma, c->sm_count, s));
    c->tvs_parity ^= 1;
    return PCT_OK;
}

extern "C" int pct_set_tvs(pct_ctx* c, float beta0, float gamma, int n_halvings) {
    if (!c) return PCT_EINVAL;
    if (!(beta0 >= 0.0f) || !isfinite(beta0)) return fail(c, PCT_EINVAL, "pct_set_tvs: beta0 must be >= 0 (0 switches the step off)");
    DeviceGuard guard(c->device);
    if (beta0 == 0.0f) {
        c->tvs_beta0 = 0.f;
        return PCT_OK;
    }
    if (!(gamma > 0.0f) || !(gamma <= 1.0f)) return fail(c, PCT_EINVAL, "pct_set_tvs: gamma must be in (0, 1]");
    if (n_halvings < 1 || n_halvings > kTvMaxLevels) return fail(c, PCT_EINVAL, "pct_set_tvs: n_halvings must be in [1, 8]");
    if (!c->tvs_grad) CUDA_TRY(c, cudaMalloc(&c->tvs_grad, sizeof(float) * c->n_slots));
    if (!c->tvs_state) CUDA_TRY(c, cudaMalloc(&c->tvs_state, sizeof(TvState)));
    TvState init{};
    init.beta[0] = init.beta[1] = beta0;
    init.beta_used = beta0;
    init.level = -1;
    CUDA_TRY(c, cudaMemcpyAsync(c->tvs_state, &init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));  // (init lives on this stack frame)
    c->tvs_beta0 = beta0;
    c->tvs_gamma = gamma;
    c->tvs_levels = n_halvings;
    c->tvs_parity = 0;
    return PCT_OK;
}

extern "C" int pct_tvs_step(pct_ctx* c) {
    if (!c) return PCT_EINVAL;
    if (!(c->tvs_beta0 > 0.0f)) return fail(c, PCT_ESTATE, "pct_tvs_step: the step is off (pct_set_tvs)");
    DeviceGuard guard(c->device);
    return tvs_step(c, c->x, c->stream);
}

extern "C" int pct_get_tvs_state(pct_ctx* c, double out[6]) {
    if (!c || !out) return PCT_EINVAL;
    if (!c->tvs_state) return fail(c, PCT_ESTATE, "pct_get_tvs_state: pct_set_tvs was never called");
    DeviceGuard guard(c->device);
    TvState h;
    CUDA_TRY(c, cudaMemcpyAsync(&h, c->tvs_state, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    out[0] = (double)h.beta[c->tvs_parity];  // the step size the next step starts from
    out[1] = h.tv_before;
    out[2] = h.tv_after;
    out[3] = (double)h.level;
    out[4] = (double)h.steps;
    out[5] = (double)h.accepted;
    return PCT_OK;
}

// The depth step of the path (R9, R33): the Sigma1^-1 table at the new node depths, the node count, the
// shared memory of the walk kernels.
extern "C" int pct_set_step(pct_ctx* c, int substeps) {
    if (!c) return PCT_EINVAL;
    if (substeps != 1 && substeps != 2) return fail(c, PCT_EINVAL, "pct_set_step: substeps must be 1 (voxel edge) or 2 (half a voxel edge)");
    DeviceGuard guard(c->device);
    const int kmax = substeps * c->g.nmin;
    if (kmax == c->g.kmax) return PCT_OK;
    int smem_max = 0;
    CUDA_TRY(c, cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
    if (((kmax + 32) >> 5) > 64 || drop_smem_bytes(kmax) + 1024 > (size_t)smem_max) {
        char what[96];
        snprintf(what, sizeof(what), "%zu B of shared memory per CTA needed, %d offered", drop_smem_bytes(kmax), smem_max);
        return fail(c, PCT_EINVAL, "pct_set_step: the grid is too wide for the half-voxel step (%s)", what);
    }
    const float step = substeps == 2 ? 0.5f * c->g.h : c->g.h;
    float4* tab = (float4*)malloc(sizeof(float4) * (kmax + 1));
    if (!tab) return fail(c, PCT_ENOMEM, "pct_set_step: out of host memory");
    sigma1_inverse_table(step, kmax, tab);
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));  // (kernels in flight still read the old table)
    cudaError_t e = cudaMemcpy(c->tab, tab, sizeof(float4) * (kmax + 1), cudaMemcpyHostToDevice);
    free(tab);
    CUDA_TRY(c, e);
    CUDA_TRY(c, drop_configure(kmax, &c->drop_grid));
    c->g.kmax = kmax;
    c->g.inv_step = 1.0f / step;
    drop_graph(c);  // the cached graph holds the old geometry
    if (c->exact_scratch) return exact_scratch_alloc(c);  // (sized by the segments a lane can own)
    return PCT_OK;
}

static int exact_scratch_alloc(pct_ctx* c) {
    if (c->exact_scratch) cudaFree(c->exact_scratch);
    c->exact_scratch = nullptr;
    // (room for 64 CTAs more than the grid: the CARP strings run side by side on ceil(grid / P) CTAs each, each with a region of its own)
    const size_t bytes = exact_scratch_bytes(c->g.kmax, c->drop_grid + 64, &c->exact_cap);
    CUDA_TRY(c, cudaMalloc(&c->exact_scratch, bytes));
    CUDA_TRY(c, exact_configure(c->g.kmax));
    return PCT_OK;
}

extern "C" int pct_set_walk(pct_ctx* c, int mode) {
    if (!c) return PCT_EINVAL;
    if (mode != PCT_WALK_MIDPOINT && mode != PCT_WALK_EXACT) return fail(c, PCT_EINVAL, "pct_set_walk: unknown mode");
    DeviceGuard guard(c->device);
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    drop_graph(c);  // the cached graph holds the other mode's kernel
    if (mode == PCT_WALK_MIDPOINT) {
        if (c->exact_scratch) cudaFree(c->exact_scratch);
        c->exact_scratch = nullptr;
        return PCT_OK;
    }
    return exact_scratch_alloc(c);
}

extern "C" int pct_set_option(pct_ctx* c, int key, int value) {
    if (!c) return PCT_EINVAL;
    switch (key) {
        case PCT_OPT_ORDER:
            if (value < 0 || value > 2) return fail(c, PCT_EINVAL, "pct_set_option: PCT_OPT_ORDER takes 0 (never), 1 (by footprint) or 2 (always)");
            c->opt_order = value;  // takes effect at the next pct_iterate / pct_iterate_carp (prepare_order)
            return PCT_OK;
        case PCT_OPT_ROWS_PAIR:
            if (value != 0 && value != 1) return fail(c, PCT_EINVAL, "pct_set_option: PCT_OPT_ROWS_PAIR takes 0 or 1");
            c->opt_rows_pair = value == 1;
            return PCT_OK;
        default:
            return fail(c, PCT_EINVAL, "pct_set_option: unknown key");
    }
}

extern "C" int pct_set_path_model(pct_ctx* c, int model) {
    if (!c) return PCT_EINVAL;
    if (model != PCT_PATH_MLP && model != PCT_PATH_SPLINE) return fail(c, PCT_EINVAL, "pct_set_path_model: unknown model");
    if (c->g.path_model != model) {
        c->g.path_model = model;
        drop_graph(c);  // the cached graph holds the kernel of the other model
    }
    return PCT_OK;
}

// Exact traversal: a history whose runs outgrow its lane's scratch is left out of its block and counted (pct_exact.cu);
// the count of the last sweep is in ctrl->last[3].  Called after the stream has been synchronised.
static const char kExactOverflow[] = "exact traversal: a path produced more runs than a lane's scratch holds (slopes beyond any tracker's); its row was left out";
static int check_exact_error(pct_ctx* c) {
    if (!c->exact_scratch) return PCT_OK;
    unsigned long long dropped = 0;
    CUDA_TRY(c, cudaMemcpyAsync(&dropped, &c->ctrl->last[3], sizeof(dropped), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return dropped ? fail(c, PCT_EINTERNAL, "%s", kExactOverflow) : PCT_OK;
}

extern "C" int pct_synchronize(pct_ctx* c) {
    if (!c) return PCT_EINVAL;
    DeviceGuard guard(c->device);
    if (int rc = wait_upload(c, -1)) return rc;  // the host arrays are free once this returns
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return check_exact_error(c);
}

extern "C" int pct_get_image(pct_ctx* c, float* dst, int64_t n_voxels) {
    if (!c) return PCT_EINVAL;
    if (!dst || n_voxels != c->n_voxels) return fail(c, PCT_EINVAL, "pct_get_image: dst NULL or n_voxels != nx*ny*nz");
    DeviceGuard guard(c->device);
    if (int rc = wait_upload(c, -1)) return rc;
    // storage order -> the caller's order, straight into dst if it is device memory
    float* out = is_device_ptr(dst) ? dst : c->io_buf;
    CUDA_TRY(c, launch_image_io(c->x, out, c->g, false, c->stream));
    if (out != dst) CUDA_TRY(c, cudaMemcpyAsync(dst, out, sizeof(float) * c->n_voxels, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return check_exact_error(c);
}

extern "C" int pct_set_image(pct_ctx* c, const float* src, int64_t n_voxels) {
    if (!c) return PCT_EINVAL;
    if (!src || n_voxels != c->n_voxels) return fail(c, PCT_EINVAL, "pct_set_image: src NULL or n_voxels != nx*ny*nz");
    DeviceGuard guard(c->device);
    const bool dev = is_device_ptr(src);
    if (!dev) CUDA_TRY(c, cudaMemcpyAsync(c->io_buf, src, sizeof(float) * c->n_voxels, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, launch_image_io(c->x, dev ? const_cast<float*>(src) : c->io_buf, c->g, true, c->stream));
    if (!dev) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return PCT_OK;
}

extern "C" int pct_image_storage(pct_ctx* c, float** image, int64_t* n_slots) {
    if (!c || !image || !n_slots) return PCT_EINVAL;
    *image = c->x;
    *n_slots = c->n_slots;
    return PCT_OK;
}

extern "C" int pct_get_stats(pct_ctx* c, int64_t out[4]) {
    if (!c || !out) return PCT_EINVAL;
    DeviceGuard guard(c->device);
    unsigned long long last[4] = {0, 0, 0, 0};
    CUDA_TRY(c, cudaMemcpyAsync(last, c->ctrl->last, sizeof(last), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < 3; ++i) out[i] = (int64_t)last[i];
    out[3] = c->n;
    if (c->exact_scratch && last[3] > 0)
        return fail(c, PCT_EINTERNAL, "%s", kExactOverflow);
    bounds_dump("pct_get_stats");
    return PCT_OK;
}

extern "C" int pct_debug_rows(pct_ctx* c, int64_t first, int64_t count, int32_t max_seg, int32_t* nseg, int32_t* nnz,
                              int32_t* seg_idx, float* seg_len, float* row_len, float* nodes) {
    if (!c) return PCT_EINVAL;
    if (!c->have_hist) return fail(c, PCT_ESTATE, "pct_debug_rows: no histories set");
    if (first < 0 || count < 1 || first + count > c->n) return fail(c, PCT_EINVAL, "pct_debug_rows: range outside the histories");
    if (max_seg < c->g.kmax + 2) return fail(c, PCT_EINVAL, "pct_debug_rows: max_seg must be >= substeps*min(nx,ny)+2");
    if (!nseg || !nnz) return fail(c, PCT_EINVAL, "pct_debug_rows: nseg and nnz are required");
    const void* outs[6] = {nseg, nnz, seg_idx, seg_len, row_len, nodes};
    for (int i = 0; i < 6; ++i)
        if (outs[i] && !is_device_ptr(outs[i])) return fail(c, PCT_EINVAL, "pct_debug_rows: outputs must be device memory");
    RowsArgs a{};
    a.g = c->g;
    a.H = c->H;
    a.first = first;
    a.count = count;
    a.max_seg = max_seg;
    a.tab = c->tab;
    a.nseg = nseg; a.nnz = nnz; a.seg_idx = seg_idx;
    a.seg_len = seg_len; a.row_len = row_len; a.nodes = nodes;
    DeviceGuard guard(c->device);
    if (int rc = wait_upload(c, first + count)) return rc;
    if (c->exact_scratch) {
        CUDA_TRY(c, launch_rows_exact(a, c->sm_count, c->stream));
        return PCT_OK;
    }
    CUDA_TRY(c, launch_rows(a, c->opt_rows_pair, c->stream));
    return PCT_OK;
}

extern "C" int pct_debug_block(pct_ctx* c, int64_t first, int64_t count, float* delta, float* cnt) {
    if (!c) return PCT_EINVAL;
    if (!c->have_hist) return fail(c, PCT_ESTATE, "pct_debug_block: no histories set");
    if (first < 0 || count < 1 || first + count > c->n) return fail(c, PCT_EINVAL, "pct_debug_block: range outside the histories");
    if (!delta || !cnt || !is_device_ptr(delta) || !is_device_ptr(cnt))
        return fail(c, PCT_EINVAL, "pct_debug_block: delta and cnt must be device memory");
    if (count > (1LL << 24)) return fail(c, PCT_EINVAL, "pct_debug_block: count must be <= 2^24 (hit counts are held exactly in fp32)");
    DeviceGuard guard(c->device);
    if (int rc = wait_upload(c, first + count)) return rc;
    CUDA_TRY(c, cudaMemsetAsync(c->ctrl, 0, sizeof(Ctrl), c->stream));
    const DropArgs a = drop_args(c, count, first, count);
    CUDA_TRY(c, launch_drop_block(a, c->drop_grid, c->stream));
    CUDA_TRY(c, launch_split_acc(c->acc, delta, cnt, c->g, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->ctrl, 0, sizeof(Ctrl), c->stream));
    return PCT_OK;
}

extern "C" int pct_debug_rule_sweep(int which, uint32_t first_bits, uint32_t last_bits, uint64_t out[2], void* cuda_stream) {
    if (!out || (which != 0 && which != 1) || first_bits > last_bits) return fail(nullptr, PCT_EINVAL, "pct_debug_rule_sweep: which must be 0 or 1, first_bits <= last_bits, out not NULL");
    unsigned long long* d = nullptr;
    const unsigned long long init[2] = {0ULL, ~0ULL};
    unsigned long long res[2] = {0ULL, 0ULL};
    cudaStream_t s = (cudaStream_t)cuda_stream;
    CUDA_TRY(nullptr, cudaMalloc(&d, sizeof(init)));
    cudaError_t e = cudaMemcpyAsync(d, init, sizeof(init), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = launch_rule_sweep(which, first_bits, last_bits, d, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(res, d, sizeof(res), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(d);
    CUDA_TRY(nullptr, e);
    out[0] = res[0];
    out[1] = res[0] ? res[1] : 0ULL;
    return PCT_OK;
}

extern "C" int pct_profile_sweep(pct_ctx* c, float lambda, int64_t block_size, float out_ms[6]) {
    if (!c) return PCT_EINVAL;
    if (!out_ms) return fail(c, PCT_EINVAL, "pct_profile_sweep: out_ms is NULL");
    if (!c->have_hist) return fail(c, PCT_ESTATE, "pct_profile_sweep: no histories set");
    if (!(lambda > 0.0f) || !(lambda < 2.0f)) return fail(c, PCT_EINVAL, "pct_profile_sweep: lambda must be in (0, 2)");
    if (block_size < 1 || block_size > (1LL << 24)) return fail(c, PCT_EINVAL, "pct_profile_sweep: block_size must be in [1, 2^24]");
    DeviceGuard guard(c->device);
    if (int rc = wait_upload(c, -1)) return rc;
    const long long n_blocks = (c->n + block_size - 1) / block_size;
    const int kChunk = 256;  // blocks per batch of events
    cudaEvent_t ev[3 * kChunk + 1];  // per block: [TVS step] accumulate, update
    int made = 0;
    int rc = PCT_OK;
    double drop_ms = 0.0, upd_ms = 0.0, tvs_ms = 0.0, total_ms = 0.0;
    const bool tvs = c->tvs_beta0 > 0.0f;
    auto body = [&]() -> int {
        for (; made < 3 * kChunk + 1; ++made) CUDA_TRY(c, cudaEventCreate(&ev[made]));
        CUDA_TRY(c, cudaMemsetAsync(c->ctrl, 0, sizeof(Ctrl), c->stream));
        prepare_order(c, block_size);
        if (int rc2 = build_order(c, block_size, n_blocks)) return rc2;
        const DropArgs a = drop_args(c, block_size, -1, 0);
        for (long long b0 = 0; b0 < n_blocks; b0 += kChunk) {
            const int nb = (int)(n_blocks - b0 < kChunk ? n_blocks - b0 : kChunk);
            CUDA_TRY(c, cudaEventRecord(ev[0], c->stream));
            for (int i = 0; i < nb; ++i) {
                if (tvs)
                    if (int rc2 = tvs_step(c, c->x, c->stream)) return rc2;
                CUDA_TRY(c, cudaEventRecord(ev[3 * i + 1], c->stream));
                CUDA_TRY(c, launch_drop_block(a, c->drop_grid, c->stream));
                CUDA_TRY(c, cudaEventRecord(ev[3 * i + 2], c->stream));
                CUDA_TRY(c, launch_update(c->x, c->acc, c->n_slots, lambda, c->ctrl, n_blocks, c->order != nullptr, c->stream));
                CUDA_TRY(c, cudaEventRecord(ev[3 * i + 3], c->stream));
            }
            CUDA_TRY(c, cudaStreamSynchronize(c->stream));
            for (int i = 0; i < nb; ++i) {
                float s = 0.f, d = 0.f, u = 0.f;
                CUDA_TRY(c, cudaEventElapsedTime(&s, ev[3 * i], ev[3 * i + 1]));
                CUDA_TRY(c, cudaEventElapsedTime(&d, ev[3 * i + 1], ev[3 * i + 2]));
                CUDA_TRY(c, cudaEventElapsedTime(&u, ev[3 * i + 2], ev[3 * i + 3]));
                tvs_ms += s;
                drop_ms += d;
                upd_ms += u;
            }
            float t = 0.f;
            CUDA_TRY(c, cudaEventElapsedTime(&t, ev[0], ev[3 * nb]));
            total_ms += t;
        }
        return PCT_OK;
    };
    rc = body();
    for (int i = 0; i < made; ++i) cudaEventDestroy(ev[i]);
    if (rc != PCT_OK) return rc;
    out_ms[0] = (float)drop_ms;
    out_ms[1] = (float)upd_ms;
    out_ms[2] = (float)total_ms;
    out_ms[4] = (float)tvs_ms;
    out_ms[5] = 0.f;
    out_ms[3] = (float)n_blocks;
    return PCT_OK;
}
