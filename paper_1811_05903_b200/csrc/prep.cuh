// prep.cuh -- row a0 of the hot path: build the j-tile records the force kernels stream.
// One CTA of TJ threads per tile; O(N) work, HBM-bound, negligible next to the O(N^2) sum.
#pragma once
#include "common.cuh"

namespace steps {

// Block-wide (min, max, max) over TJ = 256 threads; result valid in thread 0.
__device__ __forceinline__ void block_bounds(float& rlo, float& rhi, float& hh)
{
    __shared__ float s_lo[TJ / 32], s_hi[TJ / 32], s_h[TJ / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rlo = fminf(rlo, __shfl_xor_sync(0xffffffffu, rlo, o));
        rhi = fmaxf(rhi, __shfl_xor_sync(0xffffffffu, rhi, o));
        hh = fmaxf(hh, __shfl_xor_sync(0xffffffffu, hh, o));
    }
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { s_lo[w] = rlo; s_hi[w] = rhi; s_h[w] = hh; }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 1; k < TJ / 32; ++k) {
            rlo = fminf(rlo, s_lo[k]); rhi = fmaxf(rhi, s_hi[k]); hh = fmaxf(hh, s_h[k]);
        }
    }
}

template <typename Tile>
__global__ void __launch_bounds__(TJ) prep_tiles(const double* __restrict__ pos, const double* __restrict__ mass,
                                                 const double* __restrict__ soft, long long N, Tile* __restrict__ tiles)
{
    const long long j = (long long)blockIdx.x * TJ + threadIdx.x;
    const bool real = j < N;
    const double x = real ? pos[j] : STEPS_PAD_POS;
    const double y = real ? pos[N + j] : STEPS_PAD_POS;
    const double z = real ? pos[2 * N + j] : STEPS_PAD_POS;
    const double m = real ? mass[j] : 0.0;
    const double h = real ? soft[j] : 0.0;
    Tile& T = tiles[blockIdx.x];
    if constexpr (sizeof(Tile) == sizeof(TileF32)) {
        T.x[threadIdx.x] = (float)x; T.y[threadIdx.x] = (float)y; T.z[threadIdx.x] = (float)z;
        T.m[threadIdx.x] = (float)m; T.h[threadIdx.x] = (float)h;
    } else {
        T.x[threadIdx.x] = x; T.y[threadIdx.x] = y; T.z[threadIdx.x] = z;
        T.m[threadIdx.x] = m; T.h[threadIdx.x] = h;
    }
    const double r = sqrt(x * x + y * y + z * z);
    float rlo = real ? __double2float_rd(r) : __int_as_float(0x7f800000);
    float rhi = real ? __double2float_ru(r) : 0.0f;
    float hh = real ? __double2float_ru(h) : 0.0f;
    block_bounds(rlo, rhi, hh);
    if (threadIdx.x == 0) {
        T.meta.rmin = rlo; T.meta.rmax = rhi; T.meta.hmax = hh; T.meta.pad = 0.0f;
    }
}

}  // namespace steps
