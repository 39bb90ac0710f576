// common.cuh -- tile layouts, constants and small PTX helpers shared by the steps-b200 kernels.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace steps {

typedef unsigned long long u64;

// ---- decomposition constants -------------------------------------------------------------
constexpr int TJ = 256;                   // particles per j-tile (one bulk copy, one far/near decision)
constexpr int R_I = 4;                    // register-blocked i-particles per thread
constexpr int CTA_THREADS = 256;          // compute threads per CTA (8 warps)
constexpr int IB = CTA_THREADS * R_I;     // i-particles per CTA work item (1024)
constexpr int WARP_I = 32 * R_I;          // contiguous i-particles owned by one warp (128)

// Padding source: mass 0, softening 0, parked far away.  r^2 ~ 3e36 stays finite in fp32 for
// any sane |x_i|; if it overflows, rsqrt(inf) = 0 and the term is still exactly 0.
#define STEPS_PAD_POS 1.0e18

// ---- j-tile records (built by the prep kernels, streamed to shared memory as ONE bulk copy) ----
// Radial interval and largest softening of the REAL particles in the tile (pads excluded),
// rounded outwards, used for the far/near classification (triangle inequality:
// | |x_i| - |x_j| | <= |x_i - x_j|).
struct TileMeta {
    float rmin, rmax, hmax, pad;
};
struct alignas(16) TileF32 {              // mixed path: 5136 B
    float x[TJ], y[TJ], z[TJ], m[TJ], h[TJ];
    TileMeta meta;
};
struct alignas(16) TileF64 {              // fp64 path: 10256 B
    double x[TJ], y[TJ], z[TJ], m[TJ];
    double h[TJ];
    TileMeta meta;
};
static_assert(sizeof(TileF32) == 5 * TJ * 4 + 16, "TileF32 layout");
static_assert(sizeof(TileF64) == 5 * TJ * 8 + 16, "TileF64 layout");
static_assert(sizeof(TileF32) % 16 == 0 && sizeof(TileF64) % 16 == 0, "bulk copies need 16 B multiples");

// Far iff the radial gap between the i-group and the j-tile exceeds the largest possible
// pair softening, with a relative + absolute safety margin that covers the outward rounding
// of the fp32 bounds and the fp32 coordinate rounding of the mixed path (the pair law is C^1
// at r = h, so a pair within 1e-5 h of the boundary evaluated Newtonian is still exact to ~1e-10).
__device__ __forceinline__ bool tile_is_far(float rminI, float rmaxI, float hmaxI, const TileMeta& J)
{
    const float gap = fmaxf(J.rmin - rmaxI, rminI - J.rmax);
    const float need = (hmaxI + J.hmax) * 1.0001f + 1.0e-5f * fmaxf(rmaxI, J.rmax);
    return gap > need;
}

// ---- packed fp32x2 arithmetic (sm_100a FADD2 / FMUL2 / FFMA2) ------------------------------
__device__ __forceinline__ u64 pack2(float lo, float hi)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(u64 p, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p));
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b)
{
    u64 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b)
{
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c)
{
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

}  // namespace steps
