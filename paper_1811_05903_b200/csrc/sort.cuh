// sort.cuh -- row a0 of the hot path, first half: the radial order (SURVEY.md 8(a) a0 "sort by radius |x| ... when order
// changes"; the compactified sets are radially structured by construction).  The force kernels are
// correct for any order; the radial order is what makes almost every (i-group, j-tile) pair "far" (and, for the
// pair-symmetric evaluation, keeps the band of not-far block pairs narrow).  O(N log N): keys r^2 in fp64, the sort itself
// is the CUDA toolkit's device radix sort (a library primitive, not on the O(N^2) path).
#pragma once
#include <cub/device/device_radix_sort.cuh>

#include "common.cuh"

namespace steps {

__global__ void __launch_bounds__(256) radial_keys_kernel(const double* __restrict__ pos, long long N, double* __restrict__ keys,
                                                          long long* __restrict__ idx)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double x = pos[i], y = pos[N + i], z = pos[2 * N + i];
    keys[i] = fma(z, z, fma(y, y, x * x));            // >= 0: the radix order of the bit patterns is the numeric order
    idx[i] = i;
}

// dst[c][k] = src[c][perm[k]] for ncomp SoA components of length N
__global__ void __launch_bounds__(256) permute_kernel(const double* __restrict__ src, long long N, int ncomp,
                                                      const long long* __restrict__ perm, double* __restrict__ dst)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const long long j = perm[k];
    for (int c = 0; c < ncomp; ++c) dst[(long long)c * N + k] = src[(long long)c * N + j];
}

// Tile-classification statistics of the open-boundary kernels: how many (128-particle i-group, 256-source tile) pairs are
// NOT far (go through the per-pair softening test).  counts[0] += near pairs, counts[1] += all pairs.
template <typename Tile>
__global__ void __launch_bounds__(128) near_pairs_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                                                         const Tile* __restrict__ tiles, int nt, unsigned long long* __restrict__ counts)
{
    const int lane = threadIdx.x & 31;
    float rlo = __int_as_float(0x7f800000), rhi = 0.0f, hh = 0.0f;
    for (int k = threadIdx.x; k < WARP_I; k += blockDim.x) {
        const long long i = (long long)blockIdx.x * WARP_I + k;
        if (i < N) {
            const double x = pos[i], y = pos[N + i], z = pos[2 * N + i];
            const double r = sqrt(x * x + y * y + z * z);
            rlo = fminf(rlo, __double2float_rd(r)); rhi = fmaxf(rhi, __double2float_ru(r)); hh = fmaxf(hh, __double2float_ru(soft[i]));
        }
    }
    __shared__ float s_lo[4], s_hi[4], s_h[4];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rlo = fminf(rlo, __shfl_xor_sync(0xffffffffu, rlo, o)); rhi = fmaxf(rhi, __shfl_xor_sync(0xffffffffu, rhi, o));
        hh = fmaxf(hh, __shfl_xor_sync(0xffffffffu, hh, o));
    }
    if (lane == 0) { s_lo[threadIdx.x >> 5] = rlo; s_hi[threadIdx.x >> 5] = rhi; s_h[threadIdx.x >> 5] = hh; }
    __syncthreads();
    for (int w = 0; w < 4; ++w) { rlo = fminf(rlo, s_lo[w]); rhi = fmaxf(rhi, s_hi[w]); hh = fmaxf(hh, s_h[w]); }
    unsigned long long near = 0;
    for (int t = threadIdx.x; t < nt; t += blockDim.x) near += tile_is_far(rlo, rhi, hh, tiles[t].meta) ? 0 : 1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) near += __shfl_xor_sync(0xffffffffu, near, o);
    if (lane == 0) atomicAdd(&counts[0], near);
    if (threadIdx.x == 0) atomicAdd(&counts[1], (unsigned long long)nt);
}

__global__ void counts_to_double_kernel(const unsigned long long* __restrict__ counts, double* __restrict__ out2)
{
    if (threadIdx.x == 0) { out2[0] = (double)counts[0]; out2[1] = (double)counts[1]; }
}

}  // namespace steps
