// force_fp64.cuh -- pair arithmetic of the FP64 path (every pair in fp64).
//
// Rows a1/a2 of the hot path (Eq. 8 L88 first term; Eq. 3-4).
//
// Far body (scaled sources, see TileT in common.cuh): 15 FP64-pipe instructions per interaction,
// nothing else on that pipe:
//   3 DFMA  dX = X_j - c_j x_i = c_j (x_j - x_i)
//   1 DMUL + 2 DFMA  r2 = dX.dX                      (= c_j^2 r^2)
//   6 for s = r2^(-3/2) = m_j / r^3 / c_j:  y2 = y0*y0;  e = fma(-r2, y2, 1);  q3 = y0*y2;  t = q3*e;
//                      p = fma(1.875, e, 1.5);  s = fma(t, p, q3)
//   3 DFMA  acc += s * dX
// The reciprocal square root is seeded by ONE instruction on the otherwise idle SFU:
// rsqrt.approx.ftz.f64 (MUFU.RSQ64H) reads the high word of r2 and returns a double whose low
// word is zero, y0 ~ r2^(-1/2) with |delta| <~ 2^-20.  y0 has <= 21 significant bits, so y0*y0 is
// exact and e = 1 - r2*y0^2 is exact to 1e-16.  The exact factor is
//   r2^(-3/2) = y0^3 (1-e)^(-3/2) = y0^3 (1 + 1.5 e + 1.875 e^2 + 2.1875 e^3 ...);
// the body keeps the quadratic term, leaving 2.19 e^3 < 3e-18 per pair.
// Why not cheaper: a linear-only correction leaves a one-signed 1.875 e^2 ~ 1e-12 per pair whose
// pair-to-pair fluctuation is amplified by the cancellation in the net force (the bar is the MAX
// over particles, and the unluckiest of 1e6 particles has a net force ~100x below its largest
// pair terms); an fp32-computed p = 1.5 + 1.875 e has 1e-7 resolution and spoils the linear term.
// What the scaling costs: X_j = fl(c_j x_j) carries one rounding, 1.1e-16 |x_j| / r relative to
// dX -- a few 1e-15 for the closest far pairs of these sets, random in sign (measured in the
// parity tests; the unscaled 16-instruction body had exact differences).
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

// y0 ~ 1 / sqrt(r2) with ~20 good bits as an fp64 number whose low word is 0: one MUFU.RSQ64H,
// nothing on the FP64 pipe.
__device__ __forceinline__ double rsqrt_seed(double r2)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r2));
    return y;
}

// [Measured slower, kept behind STEPS_FP64_P_OFFPIPE=1 as a documented experiment: on B200 every non-FP64
//  instruction issued next to a saturated DFMA stream costs 0.3-1 clk of DFMA issue (micro-benchmark:
//  8 DFMA alone 2.37 clk each; + 4 LOP3 -> 2.84; + 4 FFMA -> 2.54), so the 6 ALU/FMA instructions that
//  replace one DFMA made the N = 1M evaluation 1224 ms instead of 1091 ms.]
// p = 1.5 + 1.875 e built WITHOUT the FP64 pipe (|e| < 2^-17; p is needed to 2^-36 absolute only,
// because it multiplies t = q3 e ~ 2^-19 q3):
//   f  = e 2^128 as an fp32 number: (hi word of e) << 3 keeps the low 8 exponent bits and the top 20
//        mantissa bits (valid for 2^-255 <= |e| < 2, and for e = 0); the sign is merged back  [SHL, LOP3]
//   g  = fma(f, 1.875 2^(38-128), 1.5 2^23): the magic-number add leaves K = rint(1.875 e 2^38) in the
//        low mantissa bits of g in two's complement, g = 0x4B400000 + K                       [FFMA]
//   p  = 1.5 + K 2^-38 as fp64 bits: (0x3FF80000'00000000 + (K << 14)); both words come straight
//        from g because 0x4B400000 is a multiple of 2^18                                     [SHF, SHF, IADD]
// Error: 2^-20 relative truncation of e (2^-39 on p) + 2^-39 rounding of K  ->  < 2^-57 relative on s.
__device__ __forceinline__ double poly_p_offpipe(double e)
{
    const unsigned H = (unsigned)__double2hiint(e);
    unsigned fb;                                               // (H << 3 & 0x7fffffff) | (H & 0x80000000): one LOP3
    asm("lop3.b32 %0, %1, %2, 0x80000000, 0xd8;" : "=r"(fb) : "r"(H << 3), "r"(H));
    const float f = __uint_as_float(fb);
    const unsigned g = __float_as_uint(fmaf(f, 0x1.ep-90f, 12582912.0f));
    const int hi = (int)(g >> 18) + (0x3ff80000 - (0x4b400000 >> 18));
    const int lo = (int)(g << 14);
    return __hiloint2double(hi, lo);
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

    // r2^(-3/2), 6 FP64-pipe instructions, relative error a few ulp.
    static __device__ __forceinline__ double rcube(double r2)
    {
        const double y0 = rsqrt_seed(r2);
        const double y2 = y0 * y0;
        const double e = fma(-r2, y2, 1.0);
        const double q3 = y0 * y2;
        const double t = q3 * e;
#if STEPS_FP64_P_OFFPIPE
        const double p = poly_p_offpipe(e);
#else
        const double p = fma(1.875, e, 1.5);
#endif
        return fma(t, p, q3);
    }

    static __device__ __forceinline__ void far(const Tile& T, const IState& S, double* acc)
    {
        double ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) ax[k] = ay[k] = az[k] = 0.0;
STEPS_UNROLL(STEPS_FAR_UNROLL)
        for (int j = 0; j < TJ; j += 2) {
            const double2 X = *reinterpret_cast<const double2*>(&T.X[j]);
            const double2 Y = *reinterpret_cast<const double2*>(&T.Y[j]);
            const double2 Z = *reinterpret_cast<const double2*>(&T.Z[j]);
            const double2 Cc = *reinterpret_cast<const double2*>(&T.c[j]);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                {
                    const double dX = fma(-S.x[k], Cc.x, X.x), dY = fma(-S.y[k], Cc.x, Y.x), dZ = fma(-S.z[k], Cc.x, Z.x);
                    const double s = rcube(fma(dZ, dZ, fma(dY, dY, dX * dX)));
                    ax[k] = fma(dX, s, ax[k]); ay[k] = fma(dY, s, ay[k]); az[k] = fma(dZ, s, az[k]);
                }
                {
                    const double dX = fma(-S.x[k], Cc.y, X.y), dY = fma(-S.y[k], Cc.y, Y.y), dZ = fma(-S.z[k], Cc.y, Z.y);
                    const double s = rcube(fma(dZ, dZ, fma(dY, dY, dX * dX)));
                    ax[k] = fma(dX, s, ax[k]); ay[k] = fma(dY, s, ay[k]); az[k] = fma(dZ, s, az[k]);
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
                double s = mq * rcube(r2);
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
