// kdk.cuh -- rows a4/a5/a7: fused kick/drift pass (Eq. 9-10, applied to
// Eq. 8) and the momentum diagnostic.  HBM-bound: 5 doubles in/out per component.
#pragma once
#include "common.cuh"

namespace steps {

struct KdkScalars {
    double ac, bc, ao, bo, gamma, B;
};

// Elementwise over the 3N components (SoA makes x/v/acc component k line up).
__global__ void __launch_bounds__(256) kick_drift_kernel(double* __restrict__ pos, double* __restrict__ vel,
                                                         const double* __restrict__ acc, long long M, KdkScalars c)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < M; k += stride) {
        const double x = pos[k];
        const double g = fma(c.B, x, acc[k]);          // acc + B x  (background term, reading #6)
        double v = vel[k];
        v = fma(c.bc, g, c.ac * v);                     // closing half kick of the previous step
        v = fma(c.bo, g, c.ao * v);                     // opening half kick of this step
        vel[k] = v;
        pos[k] = fma(c.gamma, v, x);                    // drift
    }
}

constexpr int MOM_BLOCKS = 148;

// Stage 1: fixed assignment of particles to blocks/threads, fixed-order tree -> deterministic.
__global__ void __launch_bounds__(256) momentum_stage1(const double* __restrict__ vec, const double* __restrict__ mass,
                                                        long long N, double* __restrict__ partial)
{
    double s[4] = {0, 0, 0, 0};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
        const double m = mass[i], vx = vec[i], vy = vec[N + i], vz = vec[2 * N + i];
        s[0] = fma(m, vx, s[0]); s[1] = fma(m, vy, s[1]); s[2] = fma(m, vz, s[2]);
        s[3] = fma(m, sqrt(vx * vx + vy * vy + vz * vz), s[3]);
    }
    __shared__ double sh[8][4];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_down_sync(0xffffffffu, s[c], o);
    if ((threadIdx.x & 31) == 0)
        for (int c = 0; c < 4; ++c) sh[threadIdx.x >> 5][c] = s[c];
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0;
        for (int w = 0; w < 8; ++w) t += sh[w][threadIdx.x];
        partial[blockIdx.x * 4 + threadIdx.x] = t;
    }
}

__global__ void momentum_stage2(const double* __restrict__ partial, int nblocks, double* __restrict__ out4)
{
    if (threadIdx.x < 4) {
        double t = 0;
        for (int b = 0; b < nblocks; ++b) t += partial[b * 4 + threadIdx.x];
        out4[threadIdx.x] = t;
    }
}

}  // namespace steps
