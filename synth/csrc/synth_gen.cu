// synth_gen.cu -- CUDA version of the synthetic forward model of synth/generate.py (DESIGN.md
// "Synthetic inputs"): tracker histories of a Gaussian multiple-scattering walk through an
// analytic phantom.  INPUT GENERATION ONLY: it holds none of the reconstruction's arithmetic
// (no hull, MLP, voxel walk or DROP) and is used to fill HBM with the large workloads
// (configs[2..4]) that the numpy generator would take hours to draw.  Same recipe and
// distributions as the numpy generator, different random stream (Philox keyed by (seed, i)).
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <stdint.h>

struct GenParams {
    long long first, n;
    unsigned long long seed;
    int n_angles, n_shapes, n_steps;
    float half_x, half_z, u_in;
    float wepl_noise;
    const float* shapes;  // n_shapes x 7: cx cy cz ax ay az rsp
    float *t_in, *v_in, *t_out, *v_out, *tht_in, *thv_in, *tht_out, *thv_out, *wepl;
    uint16_t* proj;
};

__global__ void __launch_bounds__(256) k_generate(const GenParams p) {
    extern __shared__ float s_shapes[];
    for (int k = threadIdx.x; k < p.n_shapes * 7; k += blockDim.x) s_shapes[k] = p.shapes[k];
    __syncthreads();
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= p.n) return;
    const long long i = p.first + r;
    curandStatePhilox4_32_10_t rng;
    curand_init(p.seed, (unsigned long long)i, 0ULL, &rng);
    const int pr = (int)(i % p.n_angles);
    double sn_d, cs_d;
    sincos(6.283185307179586 * (double)pr / (double)p.n_angles, &sn_d, &cs_d);
    const float cs = (float)cs_d, sn = (float)sn_d;
    float t = (2.0f * curand_uniform(&rng) - 1.0f) * p.half_x;
    float v = (2.0f * curand_uniform(&rng) - 1.0f) * p.half_z;
    float2 g = curand_normal2(&rng);
    float tht = 2.0e-3f * g.x, thv = 2.0e-3f * g.y;
    p.t_in[r] = t; p.v_in[r] = v; p.tht_in[r] = tht; p.thv_in[r] = thv;
    p.proj[r] = (uint16_t)pr;
    const float MP = 938.272f, X0 = 361.0f, BK_A = 0.022f, BK_P = 1.77f;
    const float r0 = BK_A * powf(200.0f, BK_P);
    float wepl = 0.0f, u = p.u_in;
    for (int s = 0; s < p.n_steps; ++s) {
        const float ds = sqrtf(1.0f + tht * tht + thv * thv);
        const float tm = t + 0.5f * tht, um = u + 0.5f, vm = v + 0.5f * thv;
        const float x = tm * cs - um * sn, y = tm * sn + um * cs, z = vm;
        float rsp = 0.001f;  // air
        for (int k = 0; k < p.n_shapes; ++k) {
            const float* q = s_shapes + 7 * k;
            const float ex = (x - q[0]) / q[3], ey = (y - q[1]) / q[4], ez = (z - q[2]) / q[5];
            if (ex * ex + ey * ey + ez * ez <= 1.0f) rsp = q[6];
        }
        wepl += rsp * ds;
        const float e = fmaxf(powf(fmaxf(r0 - wepl, 0.0f) / BK_A, 1.0f / BK_P), 1.0f);
        const float pv = (e * e + 2.0f * e * MP) / (e + MP);
        const float sig = 13.6f / pv * sqrtf(rsp * ds / X0);
        t += tht; v += thv; u += 1.0f;
        g = curand_normal2(&rng);
        tht += sig * g.x;
        thv += sig * g.y;
    }
    if (p.wepl_noise > 0.0f) wepl += p.wepl_noise * wepl * curand_normal(&rng);
    p.t_out[r] = t; p.v_out[r] = v; p.tht_out[r] = tht; p.thv_out[r] = thv; p.wepl[r] = wepl;
}

extern "C" int synth_generate(long long first, long long n, unsigned long long seed, int n_angles, int n_shapes,
                              int n_steps, float half_x, float half_z, float u_in, float wepl_noise,
                              const float* shapes_dev, float* const* out9, uint16_t* proj, void* stream) {
    if (n <= 0 || n_shapes < 0 || n_shapes > 1024) return -1;
    GenParams p;
    p.first = first; p.n = n; p.seed = seed; p.n_angles = n_angles; p.n_shapes = n_shapes; p.n_steps = n_steps;
    p.half_x = half_x; p.half_z = half_z; p.u_in = u_in; p.wepl_noise = wepl_noise; p.shapes = shapes_dev;
    p.t_in = out9[0]; p.v_in = out9[1]; p.t_out = out9[2]; p.v_out = out9[3];
    p.tht_in = out9[4]; p.thv_in = out9[5]; p.tht_out = out9[6]; p.thv_out = out9[7]; p.wepl = out9[8];
    p.proj = proj;
    const long long blocks = (n + 255) / 256;
    k_generate<<<(unsigned)blocks, 256, sizeof(float) * 7 * n_shapes, (cudaStream_t)stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}
