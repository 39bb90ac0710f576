// force_fp64.cuh -- pair arithmetic of the FP64 path (every pair in fp64).
//
// Rows a1/a2 of the hot path (Eq. 8 L88 first term; Eq. 3-4).
//
// Far body budget: 16 FP64-pipe instructions per interaction, nothing else on that pipe:
//   3 DADD  d = x_j - x_i                       (exact input differences, no cancellation loss)
//   1 DMUL + 2 DFMA  r2 = dx^2 + dy^2 + dz^2
//   7 for s = m r^-3:  y2 = y0*y0;  e = fma(-r2, y2, 1);  q = m*y0;  q3 = q*y2;  t = q3*e;
//                      c = fma(1.875, e, 1.5);  s = fma(t, c, q3)
//   3 DFMA  acc += s * d
// The reciprocal square root is seeded on the otherwise idle pipes: r2 is truncated to fp32
// with two integer ops, MUFU.RSQ gives y0 ~ r^-1 (|delta| <~ 2e-7), three integer ops widen it
// back to fp64.  With e = 1 - r2*y0^2 (exact to 1e-16: y0 has 24 bits, so y0^2 is exact) the
// exact factor is r^-3 = y0^3 (1-e)^(-3/2) = y0^3 (1 + 1.5 e + 1.875 e^2 + 2.1875 e^3 ...);
// the body keeps the quadratic term, leaving 2.19 e^3 < 3e-19 per pair.
// Why not cheaper: a linear-only correction (14 instructions) leaves a one-signed 1.875 e^2 <=
// 5e-13 per pair.  The bar is the MAX over particles, and the unluckiest of 1e6 particles has a
// net force ~100x below its largest pair terms, which amplifies any per-pair error that is
// not a few ulp; measured on config 1 the 14-instruction body gave max 4.3e-12 (rms 5e-14).
//
// Accumulation: the compactified sets put ~87 % of the mass in the outer 1 % of the particles,
// whose large pulls cancel almost exactly (shell theorem); a single running fp64 sum over all
// j reaches partial sums ~1e3 x the net force and loses ~1e-12 (measured: max 1.6e-12 on
// config 1).  So each 256-source tile is summed from zero in plain fp64 (small partials) and
// the tile result is added to a double-double (hi, lo) accumulator with an error-free TwoSum:
// 21 extra FP64 instructions per i per tile = 0.08 per interaction.
#pragma once
#include "common.cuh"

namespace steps {

// y0 ~ 1 / sqrt(r2) to fp32-SFU accuracy, as an fp64 number, without touching the FP64 pipe.
// Valid for 2^-126 <= r2 < 2^128.
__device__ __forceinline__ double rsqrt_seed(double r2)
{
    const int hi = __double2hiint(r2), lo = __double2loint(r2);
    const unsigned fb = __funnelshift_l((unsigned)lo, (unsigned)(hi - 0x38000000), 3);   // fp64 -> fp32 bits (truncate)
    const float y = rsqrt_approx(__uint_as_float(fb));
    const unsigned yb = __float_as_uint(y);
    return __hiloint2double((int)((yb >> 3) + 0x38000000u), (int)(yb << 29));            // fp32 -> fp64 bits (exact)
}

// Softened branches of Eq. 4 as g = calF / r in fp64.  Caller guarantees 0 < r2 < h^2.
__device__ __noinline__ double spline_g_soft_f64(double r2, double h)
{
    const double r = sqrt(r2);
    const double ih = 1.0 / h, u = r * ih, ih3 = ih * ih * ih;
    if (u < 0.5) return ih3 * (32.0 / 3.0 + u * u * (32.0 * u - 38.4));
    return ih3 * (64.0 / 3.0 + u * (-48.0 + u * (38.4 - (32.0 / 3.0) * u))) - 1.0 / (15.0 * r * r2);
}

struct Fp64Path {
    using Tile = TileF64;

    static constexpr int NOUT = 6;            // (hi, lo) x 3 components per i-particle

    struct IState {
        double x[R_I], y[R_I], z[R_I], h[R_I];
    };

    // acc: this thread's accumulators in shared memory; hi of component c at (c, k), lo at (3 + c, k).
    // (hi, lo) += partial with Knuth's TwoSum (error-free for any magnitudes).
    static __device__ __forceinline__ void flush(double* acc, int c, int k, double partial)
    {
        double* ph = acc + (c * R_I + k) * CTA_THREADS;
        double* pl = acc + ((3 + c) * R_I + k) * CTA_THREADS;
        const double a = *ph;
        const double s = a + partial;
        const double bb = s - a;
        const double err = (a - (s - bb)) + (partial - bb);
        *ph = s;
        *pl += err;
    }

    static __device__ __forceinline__ void load_i(IState& S, const double* __restrict__ pos,
                                                  const double* __restrict__ soft, long long N,
                                                  const long long (&idx)[R_I], float& rlo, float& rhi, float& hh)
    {
#pragma unroll
        for (int k = 0; k < R_I; ++k) {
            S.x[k] = pos[idx[k]]; S.y[k] = pos[N + idx[k]]; S.z[k] = pos[2 * N + idx[k]]; S.h[k] = soft[idx[k]];
            const double r = sqrt(S.x[k] * S.x[k] + S.y[k] * S.y[k] + S.z[k] * S.z[k]);
            rlo = fminf(rlo, __double2float_rd(r));
            rhi = fmaxf(rhi, __double2float_ru(r));
            hh = fmaxf(hh, __double2float_ru(S.h[k]));
        }
    }

    // m * r2^(-3/2), 7 FP64-pipe instructions, relative error a few ulp.
    static __device__ __forceinline__ double newton_s(double r2, double m)
    {
        const double y0 = rsqrt_seed(r2);
        const double y2 = y0 * y0;
        const double e = fma(-r2, y2, 1.0);
        const double q3 = (m * y0) * y2;
        const double t = q3 * e;
        const double c = fma(1.875, e, 1.5);
        return fma(t, c, q3);
    }

    static __device__ __forceinline__ void far(const Tile& T, const IState& S, double* acc)
    {
        double ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) ax[k] = ay[k] = az[k] = 0.0;
#pragma unroll 2
        for (int j = 0; j < TJ; j += 2) {
            const double2 X = *reinterpret_cast<const double2*>(&T.x[j]);
            const double2 Y = *reinterpret_cast<const double2*>(&T.y[j]);
            const double2 Z = *reinterpret_cast<const double2*>(&T.z[j]);
            const double2 M = *reinterpret_cast<const double2*>(&T.m[j]);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                {
                    const double dx = X.x - S.x[k], dy = Y.x - S.y[k], dz = Z.x - S.z[k];
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    const double s = newton_s(r2, M.x);
                    ax[k] = fma(dx, s, ax[k]); ay[k] = fma(dy, s, ay[k]); az[k] = fma(dz, s, az[k]);
                }
                {
                    const double dx = X.y - S.x[k], dy = Y.y - S.y[k], dz = Z.y - S.z[k];
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    const double s = newton_s(r2, M.y);
                    ax[k] = fma(dx, s, ax[k]); ay[k] = fma(dy, s, ay[k]); az[k] = fma(dz, s, az[k]);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < R_I; ++k) { flush(acc, 0, k, ax[k]); flush(acc, 1, k, ay[k]); flush(acc, 2, k, az[k]); }
    }

    static __device__ __forceinline__ void near(const Tile& T, const IState& S, double* acc)
    {
        double ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) ax[k] = ay[k] = az[k] = 0.0;
#pragma unroll 1
        for (int j = 0; j < TJ; ++j) {
            const double xj = T.x[j], yj = T.y[j], zj = T.z[j], mq = T.m[j], hj = T.h[j];
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                const double dx = xj - S.x[k], dy = yj - S.y[k], dz = zj - S.z[k];
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const double hs = S.h[k] + hj;
                double s = newton_s(r2, mq);
                if (r2 < hs * hs || r2 == 0.0)                        // Eq. 4 branches 1-2; readings #2, #4
                    s = (r2 == 0.0) ? 0.0 : mq * spline_g_soft_f64(r2, hs);
                ax[k] = fma(dx, s, ax[k]); ay[k] = fma(dy, s, ay[k]); az[k] = fma(dz, s, az[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < R_I; ++k) { flush(acc, 0, k, ax[k]); flush(acc, 1, k, ay[k]); flush(acc, 2, k, az[k]); }
    }
};

}  // namespace steps
