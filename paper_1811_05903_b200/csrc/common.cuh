// common.cuh -- tile layouts, constants and small PTX helpers shared by the steps-b200 kernels.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace steps {

typedef unsigned long long u64;

// ---- decomposition constants -------------------------------------------------------------
// (overridable with -DSTEPS_TJ / -DSTEPS_R_I / -DSTEPS_CTA_THREADS for tuning sweeps; the defaults are the product)
#ifndef STEPS_TJ
#define STEPS_TJ 256
#endif
#ifndef STEPS_R_I
#define STEPS_R_I 4
#endif
#ifndef STEPS_CTA_THREADS
#define STEPS_CTA_THREADS 512
#endif
#ifndef STEPS_FAR_UNROLL
#define STEPS_FAR_UNROLL 1
#endif
// fp64 path: far tiles summed in registers between two additions to the double-double accumulator (force_fp64.cuh)
#ifndef STEPS_FP64_FAR_TILES_PER_FLUSH
#define STEPS_FP64_FAR_TILES_PER_FLUSH 4
#endif
// Constant folded into the scaled copy of the fp64 tiles: c_j = (STEPS_FP64_FOLD m_j)^(-1/2) (force_fp64.cuh).
#define STEPS_FP64_FOLD 1.875
// fp32 tiles store c[] with adjacent elements swapped (c[j ^ 1]): after the LDS.128 loads of the far
// body the scalar c_q then sits in a register of the opposite parity (bank) to X_q / Y_q / Z_q.
#ifndef STEPS_C_SWIZZLE
#define STEPS_C_SWIZZLE 1
#endif
#define STEPS_PRAGMA_(x) _Pragma(#x)
#define STEPS_UNROLL(n) STEPS_PRAGMA_(unroll n)
constexpr int TJ = STEPS_TJ;              // particles per j-tile (one bulk copy, one far/near decision)
constexpr int R_I = STEPS_R_I;            // register-blocked i-particles per thread
constexpr int CTA_THREADS = STEPS_CTA_THREADS;   // threads per CTA; ONE persistent CTA per SM
constexpr int IB = CTA_THREADS * R_I;     // i-particles per CTA work item (2048)
constexpr int WARP_I = 32 * R_I;          // contiguous i-particles owned by one warp (128)

// Padding source: mass 0, softening 0, parked far away.  r^2 ~ 3e36 stays finite in fp32 for
// any sane |x_i|; if it overflows, rsqrt(inf) = 0 and the term is still exactly 0.
#define STEPS_PAD_POS 1.0e18
// Scaled-copy pads (and massless sources): mixed path c = 1e18, X = 1e30 (dX.dX = +inf in fp32,
// rsqrt = +0); fp64 path c = 1e100, X = 1e150 (dX.dX ~ 1e300 finite, y0 y0^2 underflows to +0).
#define STEPS_PAD_C32 1.0e18f
#define STEPS_PAD_X32 1.0e30f
#define STEPS_PAD_C64 1.0e100
#define STEPS_PAD_X64 1.0e150

// ---- j-tile records (built by the prep kernels, streamed to shared memory as ONE bulk copy) ----
// Radial interval and largest softening of the REAL particles in the tile (pads excluded),
// rounded outwards, used for the far/near classification (triangle inequality:
// | |x_i| - |x_j| | <= |x_i - x_j|).
struct TileMeta {
    float rmin, rmax, hmax, pad;
    // Axis-aligned bounding box of the REAL particles (rounded outwards), used by the periodic-box kernels: a
    // (i-group, j-tile) pair whose boxes are compact (cell-ordered input) shares ONE periodic image shift per
    // component, so the per-pair wrap of Eq. 5's leading term is only paid where the boxes straddle half the box.
    float lo[3], hi[3], pad2[2];
};
static_assert(sizeof(TileMeta) == 48, "TileMeta layout");
//
// Each tile carries its sources twice:
//   (X, Y, Z, c)    mass-scaled copy for the FAR body:  c_j = m_j^(-1/2),  X_j = c_j x_j.  With
//                   dX = X_j - c_j x_i = c_j (x_j - x_i) and y = (dX.dX)^(-1/2) = 1/(c_j r) the
//                   Newtonian term is  m_j (x_j - x_i) / r^3 = y^3 dX  -- the multiplication by
//                   m_j disappears from the pair arithmetic (11 instead of 12 FP32-pipe
//                   instructions per interaction; 15 instead of 16 on the FP64 pipe).
//   (x, y, z, m, h) plain copy for the NEAR body (per-pair softening test, Eq. 4 branches).
// Pads and massless sources have c = STEPS_PAD_C and X = STEPS_PAD_X: dX.dX overflows to +inf,
// its reciprocal square root is +0 and the term is exactly 0.
template <typename T>
struct alignas(16) TileT {
    T X[TJ], Y[TJ], Z[TJ], c[TJ];
    T x[TJ], y[TJ], z[TJ], m[TJ], h[TJ];
    TileMeta meta;
};
typedef TileT<float> TileF32;             // mixed path:  9264 B
// fp64 path, 18480 B: the scaled copy is stored per source, (X, Y, Z, c) in 32 contiguous bytes, because the
// fp64 far body handles ONE source per loop pass and every shared-memory load costs FP64-pipe issue time on
// B200 (measured: ~1.8 clk per LDS.64, ~2.5 clk per LDS.128 next to a saturated DFMA stream): two LDS.128 per
// source instead of four LDS.64.
struct alignas(16) FarSrcF64 {
    double X, Y, Z, c;
};
struct alignas(16) TileF64 {
    FarSrcF64 far[TJ];
    double x[TJ], y[TJ], z[TJ], m[TJ], h[TJ];
    TileMeta meta;
};
static_assert(sizeof(TileF32) == 9 * TJ * 4 + sizeof(TileMeta), "TileF32 layout");
static_assert(sizeof(TileF64) == 9 * TJ * 8 + sizeof(TileMeta), "TileF64 layout");
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

// ---- periodic boxes (Eq. 5, leading image): one image decision per (i-group, j-unit) pair ---------------
// With cell-ordered input the separations d = x_j - x_i of a (group, unit) pair span, per component, an interval
// [dmin, dmax] shorter than L (from the two bounding boxes).  With k = the leading-image index of dmin, i.e.
// dmin in [(k - 1/2) L, (k + 1/2) L), and top = (k + 1/2) L:
//   dmax < top    every pair takes image k:  d' = d - k L                                   (uniform shift k L)
//   otherwise     the interval holds the half-box point `top` (and, being shorter than L, no other): with e = d - top,
//                 |e| <= L, the leading image is  d' = e - copysign(L/2, e)  (image k below the point, k + 1 above it) --
//                 a FOLD: one addition and one bit operation per pair and component, no rounding to the lattice, no compare.
// The shift (k L or top) goes onto the i-particles once per (group, unit) pair (x_i' = x_i + s), so the pair arithmetic
// is the open-boundary far body plus the fold of the components in `mask`.
// gmin = the smallest |d'| any pair of the two boxes can have in this component; the pair is FAR when no separation
// can be below the largest pair softening.
// kind: 0 = a softened pair is possible, or a box pair spans a whole period (unsorted input) -> general wrapped body;
//       1 = far: shift s, fold the components in mask.
struct BoxShift {
    int kind, mask;
    double s[3];
};
__device__ __forceinline__ BoxShift box_shift(const float (&loI)[3], const float (&hiI)[3], float hmaxI, const float (&loJ)[3],
                                              const float (&hiJ)[3], float hmaxJ, double L, double invL)
{
    BoxShift d;
    d.kind = 1; d.mask = 0;
    double g2 = 0.0;
    const double eps = 1.0e-5 * L;                               // outward: fp32 rounding of the bounds and of the mixed path's coordinates
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double dmin = ((double)loJ[c] - (double)hiI[c]) - eps, dmax = ((double)hiJ[c] - (double)loI[c]) + eps;
        if (!(dmax - dmin < 0.999 * L) || !(dmax >= dmin)) { d.kind = 0; d.s[c] = 0.0; continue; }   // also NaN / inf / empty boxes
        const double k = floor(fma(dmin, invL, 0.5));
        const double top = (k + 0.5) * L;
        double gmin;
        if (dmax < top) {
            d.s[c] = k * L;
            const double lo = dmin - d.s[c], hi = dmax - d.s[c];
            gmin = lo > 0.0 ? lo : (hi < 0.0 ? -hi : 0.0);
        } else {
            d.s[c] = top; d.mask |= 1 << c;
            gmin = fmax(0.0, 0.5 * L - fmax(top - dmin, dmax - top));
        }
        g2 = fma(gmin, gmin, g2);
    }
    if (d.kind != 0) {
        const double need = ((double)hmaxI + (double)hmaxJ) * 1.0001 + eps;
        if (!(g2 > need * need)) d.kind = 0;
    }
    return d;
}
__device__ __forceinline__ BoxShift box_shift(const float (&loI)[3], const float (&hiI)[3], float hmaxI, const TileMeta& J, double L,
                                              double invL)
{
    return box_shift(loI, hiI, hmaxI, J.lo, J.hi, J.hmax, L, invL);
}

// Bounding box and largest softening of 128 consecutive particles (one i-group of the drivers; built by group_meta_kernel
// in prep.cuh), the unit of the image decisions of the pair-symmetric periodic evaluation.  An empty group (beyond N) has
// lo = +inf, hi = -inf; a group with a massless or unscalable particle has hmax = +inf (never "far").
struct alignas(16) GroupMeta {
    float lo[3], hi[3], hmax, pad;
};
static_assert(sizeof(GroupMeta) == 32, "GroupMeta layout");
// The box of GRAN consecutive groups (GRAN = 1: 128 particles, the fp64 kernels' unit; 2: 256, the mixed kernels').
template <int GRAN>
__device__ __forceinline__ GroupMeta group_box(const GroupMeta* __restrict__ gm, int idx)
{
    GroupMeta m = gm[idx * GRAN];
#pragma unroll
    for (int q = 1; q < GRAN; ++q) {
        const GroupMeta o = gm[idx * GRAN + q];
#pragma unroll
        for (int c = 0; c < 3; ++c) { m.lo[c] = fminf(m.lo[c], o.lo[c]); m.hi[c] = fmaxf(m.hi[c], o.hi[c]); }
        m.hmax = fmaxf(m.hmax, o.hmax);
    }
    return m;
}
// The image decision of the pair of groups (a, b), a != b, for separations x_j - x_i with i in a and j in b.  The boxes are
// always passed to box_shift in index order, and the decision of (b, a) is the mirror image of that of (a, b) (shift
// negated, same fold mask, same kind): the one-sided kernel (which meets every pair from both ends) and the pair-symmetric
// kernel (which meets it once) therefore agree bit for bit on which pairs "may be softened" -- each pair is evaluated by
// exactly one of them.
template <int GRAN>
__device__ __forceinline__ BoxShift pair_decision(const GroupMeta* __restrict__ gm, int a, int b, double L, double invL)
{
    const GroupMeta A = group_box<GRAN>(gm, a < b ? a : b), B = group_box<GRAN>(gm, a < b ? b : a);
    BoxShift d = box_shift(A.lo, A.hi, A.hmax, B.lo, B.hi, B.hmax, L, invL);
    if (a > b) { d.s[0] = -d.s[0]; d.s[1] = -d.s[1]; d.s[2] = -d.s[2]; }
    return d;
}

// Whether the boxes of the groups a and b span (nearly) a whole period in some component, or one of them is empty: then no
// common lattice shift centres their separations.  Boxes in index order, like pair_decision: the kernels that split the
// meetings between them by this test agree bit for bit.
template <int GRAN>
__device__ __forceinline__ bool pair_too_wide(const GroupMeta* __restrict__ gm, int a, int b, double L)
{
    const GroupMeta A = group_box<GRAN>(gm, a < b ? a : b), B = group_box<GRAN>(gm, a < b ? b : a);
    const double eps = 1.0e-5 * L;
    bool wide = false;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double dmin = ((double)B.lo[c] - (double)A.hi[c]) - eps, dmax = ((double)B.hi[c] - (double)A.lo[c]) + eps;
        wide = wide || !(dmax - dmin < 0.999 * L) || !(dmax >= dmin);
    }
    return wide;
}

// The fold of one separation component: e - copysign(h, e) as (|e| - h) with the sign of e (h = half the period, in the
// units of e).  One DADD (|e| is an operand modifier) and one LOP3 on the high word.
__device__ __forceinline__ double fold_f64(double e, double h)
{
    const double u = fabs(e) - h;
    return __hiloint2double(__double2hiint(u) ^ (__double2hiint(e) & 0x80000000), __double2loint(u));
}

// ---- Eq. 12 fused into the force evaluation's last kernel ------------------------------------------
// When `out_bits` is set, the kernel that writes the final accelerations of a FULL evaluation also forms every particle's
// step-length candidate sqrt(2 (2.8 h_i) eps / |A_i|), A_i = |G| a^-3 (acc_i + B x_i) (Eq. 12, DESIGN.md
// reading #11; a read from the device-resident run state) and folds the minimum into *out_bits with an atomicMin on the bit
// pattern (positive doubles order like their bit patterns; the minimum is exact, so the order of the atomics is immaterial).
// steps_kdk_step_adaptive uses it to skip the separate O(N) pass over (pos, acc, soft) at the start of the NEXT step.
struct Eq12Fuse {
    const double* pos;
    const double* soft;
    const double* a_state;            // &RunState::a
    double absG, B, eps;
    unsigned long long* out_bits;     // nullptr: off
};
// The candidate of one particle, exactly the arithmetic of the unfused pass (timestep_state_stage1 calls this too).
__device__ __forceinline__ double eq12_candidate(double ax, double ay, double az, double x, double y, double z, double h,
                                                 double coef, double B, double eps, double dt)
{
    const double Ax = coef * (ax + B * x);
    const double Ay = coef * (ay + B * y);
    const double Az = coef * (az + B * z);
    const double A = sqrt(Ax * Ax + Ay * Ay + Az * Az);
    if (A > 0.0) dt = fmin(dt, sqrt(2.0 * (2.8 * h) * eps / A));
    return dt;
}
__device__ __forceinline__ void eq12_fold(const Eq12Fuse& f, double dt)       // every thread of the warp calls it
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dt = fmin(dt, __shfl_xor_sync(0xffffffffu, dt, o));
    if ((threadIdx.x & 31) == 0) atomicMin(f.out_bits, (unsigned long long)__double_as_longlong(dt));
}
#define STEPS_DT_INF_BITS 0x7ff0000000000000ull

// Never-taken branch on bit n of `zero` (always 0, unknown to the compiler): ends a basic block, which
// is the only ordering ptxas respects.  One uniform-datapath branch per use, no FP64-pipe work.
#define STEPS_STAGE_FENCE(zero, n)                                                              \
    asm volatile("{\n.reg .pred p;\n.reg .b32 t;\nand.b32 t, %0, %1;\nsetp.ne.s32 p, t, 0;\n@p trap;\n}" \
                 :: "r"(zero), "r"(1 << (n)))

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
__device__ __forceinline__ u64 add2(u64 a, u64 b)
{
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
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
