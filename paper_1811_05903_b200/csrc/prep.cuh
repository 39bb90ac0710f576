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

// band_width_reset (nullable): the plan's W of a pair-symmetric evaluation (force_sym.cuh), reset here for sym_band_width.
template <typename Tile>
__global__ void __launch_bounds__(TJ) prep_tiles(const double* __restrict__ pos, const double* __restrict__ mass,
                                                 const double* __restrict__ soft, long long N, Tile* __restrict__ tiles,
                                                 int* __restrict__ band_width_reset)
{
    if (band_width_reset != nullptr && blockIdx.x == 0 && threadIdx.x == 0) *band_width_reset = 0;
    const long long j = (long long)blockIdx.x * TJ + threadIdx.x;
    const bool real = j < N;
    const double x = real ? pos[j] : STEPS_PAD_POS;
    const double y = real ? pos[N + j] : STEPS_PAD_POS;
    const double z = real ? pos[2 * N + j] : STEPS_PAD_POS;
    const double m = real ? mass[j] : 0.0;
    const double h = real ? soft[j] : 0.0;
    Tile& T = tiles[blockIdx.x];
    const int t = threadIdx.x;
    // Scaled copy (see TileT in common.cuh).  A source whose scaled coordinates would leave the
    // safe range of the arithmetic type (or with m < 0) cannot use the far body: it then forces
    // its whole tile onto the near body (hmax = +inf) -- slower, never wrong.
    bool scaled_ok = real && m > 0.0;
    if constexpr (sizeof(Tile) == sizeof(TileF32)) {
        T.x[t] = (float)x; T.y[t] = (float)y; T.z[t] = (float)z; T.m[t] = (float)m; T.h[t] = (float)h;
        // c is rounded to fp32 FIRST and X = fl32(x * c32), so that X - c32 x_i = c32 (x_j - x_i) up
        // to the one rounding of X (the same size as the fp32 rounding of x_j itself).
        const float c32 = scaled_ok ? (float)(1.0 / sqrt(m)) : STEPS_PAD_C32;
        const double lim = 1.0e18, c = (double)c32;
        scaled_ok = scaled_ok && c < lim && fabs(x * c) < lim && fabs(y * c) < lim && fabs(z * c) < lim;
        // lower end: the far body works on c r = r / sqrt(m_j) in fp32 and y^3 = (c r)^-3 must stay finite.  A far pair has
        // r >= h_i + h_j >= h_j, so c h_j bounds c r from below (h_j = 0: the documented domain of steps.h applies).
        scaled_ok = scaled_ok && !(h > 0.0 && c * h < 1.0e-12);
        T.c[t ^ STEPS_C_SWIZZLE] = scaled_ok ? c32 : STEPS_PAD_C32;   // see STEPS_C_SWIZZLE in common.cuh
        T.X[t] = scaled_ok ? (float)(x * c) : STEPS_PAD_X32;
        T.Y[t] = scaled_ok ? (float)(y * c) : STEPS_PAD_X32;
        T.Z[t] = scaled_ok ? (float)(z * c) : STEPS_PAD_X32;
    } else {
        T.x[t] = x; T.y[t] = y; T.z[t] = z; T.m[t] = m; T.h[t] = h;
        // c_j = (1.875 m_j)^(-1/2): the fp64 far body returns s = r2^(-3/2) / 1.875 (force_fp64.cuh), so that
        // s dX = c_j^-2 (x_j - x_i) / (1.875 r^3) = m_j (x_j - x_i) / r^3
        const double lim = 1.0e100, c = scaled_ok ? 1.0 / sqrt(STEPS_FP64_FOLD * m) : STEPS_PAD_C64;
        scaled_ok = scaled_ok && c < lim && fabs(x * c) < lim && fabs(y * c) < lim && fabs(z * c) < lim;
        T.far[t].c = scaled_ok ? c : STEPS_PAD_C64;
        T.far[t].X = scaled_ok ? x * c : STEPS_PAD_X64;
        T.far[t].Y = scaled_ok ? y * c : STEPS_PAD_X64;
        T.far[t].Z = scaled_ok ? z * c : STEPS_PAD_X64;
    }
    // A massless particle exerts nothing either way (its scaled copy is parked), but as a TARGET of the pair-symmetric
    // evaluation its reaction sum could not be divided by m_j: its tile is marked like an unscalable one, which keeps every
    // block pair of its block out of the symmetric items (W = nb - 1 on the device).
    const bool force_near = real && !scaled_ok;
    const double r = sqrt(x * x + y * y + z * z);
    float rlo = real ? __double2float_rd(r) : __int_as_float(0x7f800000);
    float rhi = real ? __double2float_ru(r) : 0.0f;
    float hh = real ? __double2float_ru(h) : 0.0f;
    if (force_near) hh = __int_as_float(0x7f800000);
    block_bounds(rlo, rhi, hh);
    if (threadIdx.x == 0) {
        T.meta.rmin = rlo; T.meta.rmax = rhi; T.meta.hmax = hh; T.meta.pad = 0.0f; T.meta.pad2[0] = T.meta.pad2[1] = 0.0f;
    }
    // bounding box (three more rounds of the same reduction; prep is O(N) and < 0.01 % of an evaluation)
    const float inf = __int_as_float(0x7f800000);
    const double cs[3] = {x, y, z};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        __syncthreads();                                     // block_bounds' shared scratch is reused
        float lo = real ? __double2float_rd(cs[c]) : inf, hi = real ? __double2float_ru(cs[c]) : -inf, unused = 0.0f;
        block_bounds(lo, hi, unused);
        if (threadIdx.x == 0) { T.meta.lo[c] = lo; T.meta.hi[c] = hi; }
    }
}

// Bounding box and largest softening of every group of 128 consecutive particles (GroupMeta, common.cuh); one warp per
// group, `ngroups` >= ceil(N / 128) (the groups beyond N are written empty).  Runs after prep_tiles: a tile that prep
// marked hmax = +inf (a massless or unscalable particle) passes the mark on to its two groups.
template <typename Tile>
__global__ void __launch_bounds__(128) group_meta_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                                                         const Tile* __restrict__ tiles, GroupMeta* __restrict__ gm, int ngroups)
{
    const int g = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (g >= ngroups) return;
    const float inf = __int_as_float(0x7f800000);
    float lo[3] = {inf, inf, inf}, hi[3] = {-inf, -inf, -inf}, hh = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const long long i = (long long)g * 128 + lane + 32 * k;
        if (i < N) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double v = pos[c * N + i];
                lo[c] = fminf(lo[c], __double2float_rd(v)); hi[c] = fmaxf(hi[c], __double2float_ru(v));
            }
            hh = fmaxf(hh, __double2float_ru(soft[i]));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o)); hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
        }
        hh = fmaxf(hh, __shfl_xor_sync(0xffffffffu, hh, o));
    }
    if (lane == 0) {
        if ((long long)g * 128 < N) hh = fmaxf(hh, tiles[g / 2].meta.hmax >= inf ? inf : 0.0f);
        GroupMeta m;
#pragma unroll
        for (int c = 0; c < 3; ++c) { m.lo[c] = lo[c]; m.hi[c] = hi[c]; }
        m.hmax = hh; m.pad = 0.0f;
        gm[g] = m;
    }
}

}  // namespace steps
