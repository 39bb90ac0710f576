// force_v1.cuh -- simple force driver: one CTA per 1024-particle i-block, every j-tile copied
// to shared memory with plain loads and __syncthreads.  Kept as the in-library cross-check
// of the persistent TMA driver (steps_forces_range_v1 in steps_internal.h; tests only).
#pragma once
#include "common.cuh"

namespace steps {

template <typename Path>
__global__ void __launch_bounds__(CTA_THREADS, 2)
forces_v1_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                 const typename Path::Tile* __restrict__ tiles, int ntiles,
                 long long i_begin, long long i_end, double* __restrict__ acc_out)
{
    using Tile = typename Path::Tile;
    __shared__ Tile tile;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long i0 = i_begin + (long long)blockIdx.x * IB + (long long)warp * WARP_I + lane;
    long long idx[R_I];
#pragma unroll
    for (int k = 0; k < R_I; ++k) {
        const long long i = i0 + 32 * k;
        idx[k] = i < i_end ? i : i_end - 1;
    }
    typename Path::IState S;
    float rlo = __int_as_float(0x7f800000), rhi = 0.0f, hh = 0.0f;
    Path::load_i(S, pos, soft, N, idx, rlo, rhi, hh);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rlo = fminf(rlo, __shfl_xor_sync(0xffffffffu, rlo, o));
        rhi = fmaxf(rhi, __shfl_xor_sync(0xffffffffu, rhi, o));
        hh = fmaxf(hh, __shfl_xor_sync(0xffffffffu, hh, o));
    }
    for (int t = 0; t < ntiles; ++t) {
        __syncthreads();
        {
            const uint4* src = reinterpret_cast<const uint4*>(tiles + t);
            uint4* dst = reinterpret_cast<uint4*>(&tile);
            for (int q = threadIdx.x; q < (int)(sizeof(Tile) / 16); q += CTA_THREADS) dst[q] = src[q];
        }
        __syncthreads();
        if (tile_is_far(rlo, rhi, hh, tile.meta)) Path::far(tile, S);
        else Path::near(tile, S);
    }
    const long long cnt = i_end - i_begin;
#pragma unroll
    for (int k = 0; k < R_I; ++k) {
        const long long i = i0 + 32 * k;
        if (i < i_end) {
            acc_out[i - i_begin] = S.ax[k];
            acc_out[cnt + (i - i_begin)] = S.ay[k];
            acc_out[2 * cnt + (i - i_begin)] = S.az[k];
        }
    }
}

}  // namespace steps
