// pct_noalloc.cu -- pct_tvs_step_static: one total-variation superiorization step (R31) that
// never asks the CUDA runtime for memory.
//
// Who needs this.  The regular route to a TVS step, pct_create + pct_set_tvs + pct_tvs_step, calls cudaMalloc three
// times (the context's image, the gradient array, the step's state block).  That is fine at start-up, and impossible for
// some programs later on:
//   * a host application that handed ALL device memory to an allocator of its own when it started (a framework's caching
//     pool, a fixed partition of the GPU between services of a treatment-planning system): a cudaMalloc issued from
//     inside a library then fails, or succeeds only by taking memory the application believes it owns;
//   * a reconstruction loop with a latency bound (the "real-time" of the paper's title): cudaMalloc and cudaFree
//     synchronise the whole device, so one allocation in a side computation stalls every other stream for its duration;
//   * code whose device-memory use is fixed and audited before it is allowed to run, where an allocation whose size
//     depends on a run-time argument is not acceptable.
// For such callers the step's working memory -- the image in the library's 2 x 2-tiled storage order, the gradient of TV
// and the sums of the step -- lives in a file-scope __device__ array of fixed size.  It is part of the library's device
// image: EVERY GPU on which this library's kernels get loaded holds these 8 MiB + 256 B from then until the process ends,
// whether or not this entry point is ever called.  That is the price, and the reason for the modest limit
// PCT_TVS_STATIC_MAX_SLOTS.
//
// The stencil kernels are the ones of pct_tvs.cu (launch_tvs_step), unchanged; what is new here are the two kernels that
// move the caller's image into and out of the static array (they name the array directly, as device code may) and the
// host-side set-up.  In host code the array's name is only a handle: the address a kernel argument needs comes from
// cudaGetSymbolAddress, asked once per device with that device current, and is kept per device.
#include <math.h>
#include <stdio.h>

#include <mutex>

#include "../../include/pct.h"
#include "pct_internal.h"

namespace {

using pct::Geom;
using pct::TvState;

constexpr long long kMaxSlots = PCT_TVS_STATIC_MAX_SLOTS;
constexpr size_t kStateBytes = 256;  // the state block, padded so that both float arrays start on a 256 B boundary
static_assert(sizeof(TvState) <= kStateBytes, "TvState must fit the first 256 B of the static scratch");
constexpr size_t kImageOff = kStateBytes;
constexpr size_t kGradOff = kImageOff + sizeof(float) * kMaxSlots;
constexpr size_t kScratchBytes = kGradOff + sizeof(float) * kMaxSlots;

// The scratch.  Shared by every call on a device; it keeps whatever the last call left in it.
static __device__ __align__(256) unsigned char g_tvs_scratch[kScratchBytes];

__device__ __forceinline__ TvState* scratch_state() { return reinterpret_cast<TvState*>(g_tvs_scratch); }
__device__ __forceinline__ float* scratch_image() { return reinterpret_cast<float*>(g_tvs_scratch + kImageOff); }

// Caller's image (i + nx (j + ny k)) -> storage order in the scratch.  Every one of the n_slots entries this call will
// read is written: the padding of odd grids must be zero for the stencils, and the previous call (maybe of a larger or
// differently shaped grid) left its own values there.  The state block is started from zero as well: its sums are
// accumulated with atomics, stale sums would be added to.
__global__ void k_static_stage_in(const float* __restrict__ image, Geom g, long long n_slots, float beta) {
    float* x = scratch_image();
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n_slots; s += stride) {
        int i, j, k;
        pct::voxel_of_slot((int)s, g.nxp, g.slice_p, i, j, k);
        x[s] = (i < g.nx && j < g.ny) ? __ldg(image + (i + (long long)g.nx * (j + (long long)g.ny * k))) : 0.f;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        TvState init{};  // all sums, counters zero
        init.beta[0] = init.beta[1] = beta;
        init.beta_used = beta;
        init.level = -1;
        *scratch_state() = init;
    }
}

// ... and back, plus the step's report.
__global__ void k_static_stage_out(float* __restrict__ image, Geom g, double* __restrict__ info) {
    const float* x = scratch_image();
    const long long n = (long long)g.nx * g.ny * g.nz;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const int i = (int)(v % g.nx), j = (int)((v / g.nx) % g.ny), k = (int)(v / ((long long)g.nx * g.ny));
        image[v] = x[pct::voxel_slot(i, j, k, g.nxp, g.slice_p)];
    }
    if (info && blockIdx.x == 0 && threadIdx.x == 0) {
        const TvState* st = scratch_state();
        info[0] = (double)st->beta_used;
        info[1] = st->tv_before;
        info[2] = st->tv_after;
        info[3] = (double)st->level;
    }
}

// Per-device set-up: the scratch's device address and the SM count.
constexpr int kMaxDevices = 64;
struct DeviceSetup {
    bool ready = false;
    unsigned char* base = nullptr;
    int sms = 0;
};
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;
thread_local char g_err[320] = {0};

int fail(int code, const char* fmt, const char* detail = "") {
    snprintf(g_err, sizeof(g_err), fmt, detail);
    return code;
}

bool on_device(const void* p, int dev) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeManaged || (at.type == cudaMemoryTypeDevice && at.device == dev);
}

}  // namespace

extern "C" const char* pct_tvs_step_static_error(void) { return g_err; }

extern "C" int pct_tvs_step_static(float* image, int nx, int ny, int nz, float beta, int n_halvings, double* info, void* cuda_stream) {
    // argument checks first: they need no GPU and touch no CUDA state
    if (!image) return fail(PCT_EINVAL, "pct_tvs_step_static: image is NULL");
    if (nx < 1 || ny < 1 || nz < 1) return fail(PCT_EINVAL, "pct_tvs_step_static: grid dimensions must be >= 1");
    const long long nxp = ((long long)nx + 1) & ~1LL, nyp = ((long long)ny + 1) & ~1LL;
    const long long n_slots = nxp * nyp * nz;
    if (n_slots > kMaxSlots) {
        char what[160];
        snprintf(what, sizeof(what), "%d x %d x %d is stored as %lld voxels (nx, ny rounded up to even), the static scratch holds %lld",
                 nx, ny, nz, n_slots, kMaxSlots);
        return fail(PCT_EINVAL, "pct_tvs_step_static: grid too large: %s; use pct_set_tvs / pct_tvs_step on a context instead", what);
    }
    if (!(beta > 0.0f) || !isfinite(beta)) return fail(PCT_EINVAL, "pct_tvs_step_static: beta must be positive and finite");
    if (n_halvings < 1 || n_halvings > pct::kTvMaxLevels) return fail(PCT_EINVAL, "pct_tvs_step_static: n_halvings must be in [1, 8]");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(PCT_ECUDA, "pct_tvs_step_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(PCT_EINVAL, "pct_tvs_step_static: device ordinal beyond 63");
    if (!on_device(image, dev)) return fail(PCT_EINVAL, "pct_tvs_step_static: image must be device memory of the current device");
    if (info && !on_device(info, dev)) return fail(PCT_EINVAL, "pct_tvs_step_static: info must be NULL or device memory of the current device");

    DeviceSetup su;
    {
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        DeviceSetup& d = g_setup[dev];
        if (!d.ready) {  // first call on this device (it is current): ask where the array lives HERE
            unsigned char* base = nullptr;
            e = cudaGetSymbolAddress((void**)&base, g_tvs_scratch);
            if (e != cudaSuccess || !base)
                return fail(PCT_ECUDA, "pct_tvs_step_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess) return fail(PCT_ECUDA, "pct_tvs_step_static: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
            d.base = base;
            d.sms = sms;
            d.ready = true;
        }
        su = d;
    }

    Geom g{};  // the stencil and staging kernels read only the grid's extent and its storage strides
    g.nx = nx, g.ny = ny, g.nz = nz, g.nmin = nx < ny ? nx : ny;
    g.nxp = (int)nxp;
    g.slice_p = (int)(nxp * nyp);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    TvState* st = reinterpret_cast<TvState*>(su.base);
    float* x = reinterpret_cast<float*>(su.base + kImageOff);
    float* grad = reinterpret_cast<float*>(su.base + kGradOff);

    long long blocks = (n_slots + 255) / 256;
    const long long cap = (long long)su.sms * 16;
    if (blocks > cap) blocks = cap;
    k_static_stage_in<<<(int)blocks, 256, 0, stream>>>(image, g, n_slots, beta);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = pct::launch_tvs_step(x, grad, g, n_slots, st, /*parity=*/0, n_halvings, /*gamma=*/1.0f, su.sms, stream);
    if (e == cudaSuccess) {
        k_static_stage_out<<<(int)blocks, 256, 0, stream>>>(image, g, info);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return fail(PCT_ECUDA, "pct_tvs_step_static: kernel launch: %s", cudaGetErrorString(e));
    return PCT_OK;
}
