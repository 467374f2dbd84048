// pct_peaks.cu -- micro-benchmarks that give the DENOMINATORS of the metric's roofline (SURVEY.md 8(d):
// "measure: random 4 B gather ... red.global.add.f32 to uniformly random addresses in an L2-resident array",
// "fp32 issue rate").  The hot path gathers x (4 B per path segment) and reduces (Delta, c) (8 B per non-zero)
// at data-dependent addresses of an array the size of image + accumulator; what the memory system of THIS GPU
// sustains for exactly those two access kinds, and what the SMs sustain for the packed / scalar fp32 FMA the
// rule is made of, is measured here with hand-written kernels and CUDA events.  Not part of the path.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pct.h"

namespace pctpeaks {

__device__ __forceinline__ uint32_t next_rand(uint32_t& s) {  // xorshift32
    s ^= s << 13;
    s ^= s >> 17;
    s ^= s << 5;
    return s;
}
__device__ __forceinline__ uint32_t seed_of(uint32_t tid) {
    uint32_t s = tid * 2654435761u + 0x9e3779b9u;
    s ^= s >> 15;
    s *= 0x85ebca6bu;
    s ^= s >> 13;
    return s | 1u;
}

constexpr int kIlp = 8;  // independent requests a thread has in flight

// Every lane of every request at its own uniformly random word of the footprint: one 32 B sector per lane.
__global__ void __launch_bounds__(256) k_gather_random(const float* __restrict__ buf, uint32_t n_words, int iters, float* sink) {
    uint32_t s = seed_of(blockIdx.x * blockDim.x + threadIdx.x);
    float acc = 0.f;
    for (int it = 0; it < iters; ++it) {
        float v[kIlp];
#pragma unroll
        for (int u = 0; u < kIlp; ++u) {
            const uint32_t idx = (uint32_t)(((uint64_t)next_rand(s) * n_words) >> 32);
            v[u] = __ldcg(buf + idx);
        }
#pragma unroll
        for (int u = 0; u < kIlp; ++u) acc += v[u];
    }
    if (acc == 123.456f) *sink = acc;
}

// The path's access shape: the 32 lanes of a request touch 32 voxels one voxel apart along a random in-plane
// direction of a volume nx x nx x nz words (nx a power of two), as the segment-major passes of the row projection
// do: neighbouring lanes share a 32 B sector when the direction is close to the x axis.
template <bool TILED>
__device__ __forceinline__ uint32_t path_index(uint32_t& s, int lane, int nx, int nz) {
    const uint32_t r0 = next_rand(s), r1 = next_rand(s);
    const float ax = (float)(r0 & 63u) - 31.5f, ay = (float)((r0 >> 6) & 63u) - 31.5f;
    const float inv = rsqrtf(ax * ax + ay * ay) * (float)lane;
    const int xi = ((int)(r0 >> 12) + __float2int_rn(ax * inv)) & (nx - 1);
    const int yi = ((int)(r1 & 0xffffu) + __float2int_rn(ay * inv)) & (nx - 1);
    const uint32_t z = (uint32_t)(((uint64_t)(r1 >> 16) * (uint32_t)nz) >> 16);
    if (TILED)  // 2 x 2 in-plane tiles, two x-adjacent tiles side by side: a 32 B sector = 4 x 2 words or 2 x 2 pairs
        return z * (uint32_t)nx * (uint32_t)nx + ((((uint32_t)yi >> 1) * ((uint32_t)nx >> 1) + ((uint32_t)xi >> 1)) << 2) +
               (((uint32_t)yi & 1u) << 1) + ((uint32_t)xi & 1u);
    return (z * (uint32_t)nx + (uint32_t)yi) * (uint32_t)nx + (uint32_t)xi;
}

template <bool TILED>
__global__ void __launch_bounds__(256) k_gather_paths(const float* __restrict__ buf, int nx, int nz, int iters, float* sink) {
    const int lane = threadIdx.x & 31;
    uint32_t s = seed_of((blockIdx.x * blockDim.x + threadIdx.x) >> 5);  // warp-uniform stream
    float acc = 0.f;
    for (int it = 0; it < iters; ++it) {
        float v[kIlp];
#pragma unroll
        for (int u = 0; u < kIlp; ++u) v[u] = __ldcg(buf + path_index<TILED>(s, lane, nx, nz));
#pragma unroll
        for (int u = 0; u < kIlp; ++u) acc += v[u];
    }
    if (acc == 123.456f) *sink = acc;
}

template <bool TILED>
__global__ void __launch_bounds__(256) k_red_paths(float2* __restrict__ buf, int nx, int nz, int iters) {
    const int lane = threadIdx.x & 31;
    uint32_t s = seed_of((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kIlp; ++u)
            asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(buf + path_index<TILED>(s, lane, nx, nz)), "f"(1.0f), "f"(1.0f) : "memory");
    }
}

// The kernel's own mix: one path-shaped gather from the image and one path-shaped vector reduction into the accumulator
// per segment (two arrays, image : accumulator = 1 : 2 of the footprint), issued back to back like the row passes.
template <bool TILED>
__global__ void __launch_bounds__(256) k_mixed_paths(const float* __restrict__ img, float2* __restrict__ acc, int nx, int nz, int iters,
                                                     float* sink) {
    const int lane = threadIdx.x & 31;
    uint32_t s = seed_of((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    float sum = 0.f;
    for (int it = 0; it < iters; ++it) {
        float v[kIlp];
        uint32_t idx[kIlp];
#pragma unroll
        for (int u = 0; u < kIlp; ++u) {
            idx[u] = path_index<TILED>(s, lane, nx, nz);
            v[u] = __ldcg(img + idx[u]);
        }
#pragma unroll
        for (int u = 0; u < kIlp; ++u) {
            sum += v[u];
            asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(acc + idx[u]), "f"(1.0f), "f"(1.0f) : "memory");
        }
    }
    if (sum == 123.456f) *sink = sum;
}

__global__ void __launch_bounds__(256) k_red_random(float2* __restrict__ buf, uint32_t n_pairs, int iters) {
    uint32_t s = seed_of(blockIdx.x * blockDim.x + threadIdx.x);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kIlp; ++u) {
            const uint32_t idx = (uint32_t)(((uint64_t)next_rand(s) * n_pairs) >> 32);
            asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(buf + idx), "f"(1.0f), "f"(1.0f) : "memory");
        }
    }
}

__global__ void __launch_bounds__(256) k_stream_read(const float4* __restrict__ buf, size_t n4, float* sink) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    float acc = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += 4 * stride) {
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = i + u * stride < n4 ? __ldcg(buf + i + u * stride) : make_float4(0, 0, 0, 0);
#pragma unroll
        for (int u = 0; u < 4; ++u) acc += v[u].x + v[u].y + v[u].z + v[u].w;
    }
    if (acc == 123.456f) *sink = acc;
}

__global__ void __launch_bounds__(256) k_ffma(int iters, float* sink) {
    float a[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) a[u] = (float)(threadIdx.x + u);
    const float m = 1.0000001f, c = 1e-9f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int u = 0; u < 8; ++u) a[u] = __fmaf_rn(a[u], m, c);
    }
    float t = 0.f;
#pragma unroll
    for (int u = 0; u < 8; ++u) t += a[u];
    if (t == 123.456f) *sink = t;
}

__global__ void __launch_bounds__(256) k_ffma2(int iters, float* sink) {
    unsigned long long a[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) asm("mov.b64 %0, {%1, %2};" : "=l"(a[u]) : "f"((float)(threadIdx.x + u)), "f"((float)u));
    unsigned long long m, c;
    asm("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(1.0000001f));
    asm("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(1e-9f));
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int u = 0; u < 8; ++u) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[u]) : "l"(m), "l"(c));
    }
    unsigned long long t = 0;
#pragma unroll
    for (int u = 0; u < 8; ++u) t ^= a[u];
    if (t == 0x123456789abcdefULL) *sink = 1.f;
}

}  // namespace pctpeaks

using namespace pctpeaks;

namespace {
struct Timer {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaStream_t s;
    explicit Timer(cudaStream_t st) : s(st) {
        cudaEventCreate(&e0);
        cudaEventCreate(&e1);
    }
    ~Timer() {
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    }
    void start() { cudaEventRecord(e0, s); }
    double stop_ms() {
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        return (double)ms;
    }
};
}  // namespace

extern "C" int pct_measure_peaks(void* stream, int64_t footprint_bytes, double out[12]) {
    if (!out || footprint_bytes < (1 << 20) || footprint_bytes > (1LL << 34)) return PCT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PCT_ECUDA;
    const size_t bytes = ((size_t)footprint_bytes / 1024) * 1024;
    float* buf = nullptr;
    float* sink = nullptr;
    if (cudaMalloc(&buf, bytes) != cudaSuccess || cudaMalloc(&sink, 64) != cudaSuccess) {
        if (buf) cudaFree(buf);
        (void)cudaGetLastError();
        return PCT_ENOMEM;
    }
    cudaMemsetAsync(buf, 0, bytes, st);
    const uint32_t n_words = (uint32_t)(bytes / 4), n_pairs = (uint32_t)(bytes / 8);
    const int grid = sms * 8;
    const double threads = (double)grid * 256.0;
    Timer T(st);
    // random 4 B gather
    const int it_g = 256;
    k_gather_random<<<grid, 256, 0, st>>>(buf, n_words, it_g, sink);  // warm-up: the footprint is in the L2 if it fits
    T.start();
    k_gather_random<<<grid, 256, 0, st>>>(buf, n_words, it_g, sink);
    double ms = T.stop_ms();
    out[0] = threads * it_g * kIlp / (ms * 1e-3);  // loads/s (one 32 B sector each)
    // path-shaped gather: the largest volume nx x nx x nz words (nx a power of two <= 256) inside the footprint
    int nx = 256;
    while ((uint64_t)nx * nx * 4 > n_words && nx > 16) nx >>= 1;
    const int nz_g = (int)(n_words / ((uint32_t)nx * nx));
    k_gather_paths<false><<<grid, 256, 0, st>>>(buf, nx, nz_g, it_g, sink);
    T.start();
    k_gather_paths<false><<<grid, 256, 0, st>>>(buf, nx, nz_g, it_g, sink);
    ms = T.stop_ms();
    out[1] = threads * it_g * kIlp / (ms * 1e-3);
    T.start();
    k_gather_paths<true><<<grid, 256, 0, st>>>(buf, nx, nz_g, it_g, sink);
    ms = T.stop_ms();
    out[8] = threads * it_g * kIlp / (ms * 1e-3);
    // random 8 B vector reduction
    const int it_r = 128;
    k_red_random<<<grid, 256, 0, st>>>((float2*)buf, n_pairs, it_r);
    T.start();
    k_red_random<<<grid, 256, 0, st>>>((float2*)buf, n_pairs, it_r);
    ms = T.stop_ms();
    out[2] = threads * it_r * kIlp / (ms * 1e-3);  // reductions/s
    // path-shaped 8 B vector reduction
    const int nz_r = (int)(n_pairs / ((uint32_t)nx * nx));
    k_red_paths<false><<<grid, 256, 0, st>>>((float2*)buf, nx, nz_r > 0 ? nz_r : 1, it_r);
    T.start();
    k_red_paths<false><<<grid, 256, 0, st>>>((float2*)buf, nx, nz_r > 0 ? nz_r : 1, it_r);
    ms = T.stop_ms();
    out[6] = threads * it_r * kIlp / (ms * 1e-3);
    T.start();
    k_red_paths<true><<<grid, 256, 0, st>>>((float2*)buf, nx, nz_r > 0 ? nz_r : 1, it_r);
    ms = T.stop_ms();
    out[9] = threads * it_r * kIlp / (ms * 1e-3);
    // streaming 128-bit reads of the footprint
    k_stream_read<<<grid, 256, 0, st>>>((const float4*)buf, bytes / 16, sink);
    T.start();
    for (int r = 0; r < 8; ++r) k_stream_read<<<grid, 256, 0, st>>>((const float4*)buf, bytes / 16, sink);
    ms = T.stop_ms();
    out[3] = 8.0 * (double)bytes / (ms * 1e-3);  // B/s
    // fp32 issue rate: scalar FMA and packed FMA (thread-instructions/s)
    const int it_f = 4096;
    k_ffma<<<grid, 256, 0, st>>>(64, sink);
    T.start();
    k_ffma<<<grid, 256, 0, st>>>(it_f, sink);
    ms = T.stop_ms();
    out[4] = threads * it_f * 64.0 / (ms * 1e-3);
    k_ffma2<<<grid, 256, 0, st>>>(64, sink);
    T.start();
    k_ffma2<<<grid, 256, 0, st>>>(it_f, sink);
    ms = T.stop_ms();
    out[5] = threads * it_f * 64.0 / (ms * 1e-3);  // packed instructions/s (two FMAs each)
    out[7] = (double)bytes;
    // the mix of the kernel: image (a third of the footprint) gathered, accumulator (two thirds) reduced, same voxel
    {
        const int nz_m = (int)(n_words / 3 / ((uint32_t)nx * nx));
        const float* img = buf;
        float2* acc = (float2*)(buf + (size_t)nx * nx * (nz_m > 0 ? nz_m : 1));
        k_mixed_paths<true><<<grid, 256, 0, st>>>(img, acc, nx, nz_m > 0 ? nz_m : 1, it_r, sink);
        T.start();
        k_mixed_paths<true><<<grid, 256, 0, st>>>(img, acc, nx, nz_m > 0 ? nz_m : 1, it_r, sink);
        ms = T.stop_ms();
        out[10] = threads * it_r * kIlp / (ms * 1e-3);  // (gather + reduction) pairs per second
    }
    out[11] = 0.0;
    cudaError_t e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaFree(buf);
    cudaFree(sink);
    return e == cudaSuccess ? PCT_OK : PCT_ECUDA;
}
