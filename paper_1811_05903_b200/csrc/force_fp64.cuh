// force_fp64.cuh -- pair arithmetic of the FP64 path (every pair in fp64).
//
// Rows a1/a2 of the hot path (Eq. 8 L88 first term; Eq. 3-4).
//
// Far body (scaled sources, see TileT in common.cuh): 14 FP64-pipe instructions per interaction,
// nothing else on that pipe:
//   3 DFMA  dX = X_j - c_j x_i = c_j (x_j - x_i)          (c_j = (1.875 m_j)^(-1/2), see below)
//   1 DMUL + 2 DFMA  r2 = dX.dX                            (= c_j^2 r^2)
//   5 for s = r2^(-3/2) / 1.875:   y2 = y0*y0;  w = fma(r2, y2, -1.4);  g = fma(w, w, C0);
//                                  q3 = y0*y2;  s = q3*g
//   3 DFMA  acc += s * dX
// The reciprocal square root is seeded by ONE instruction on the otherwise idle SFU:
// rsqrt.approx.ftz.f64 (MUFU.RSQ64H) reads the high word of r2 and returns a double whose low
// word is zero, y0 ~ r2^(-1/2) with |1 - r2 y0^2| = |e| <= 2^-19.05 (measured over 1.6e7 arguments).
// y0 has <= 21 significant bits, so y2 = y0*y0 is exact.  With u = r2 y0^2 = 1 - e the exact factor is
//   r2^(-3/2) = y0^3 u^(-3/2) = y0^3 (1 + 1.5 e + 1.875 e^2 + 2.1875 e^3 ...)
// and the quadratic Taylor polynomial 4.375 - 5.25 u + 1.875 u^2 completes to the square
//   1.875 [ (u - 1.4)^2 + 0.7/1.875 ],
// which costs two FMAs (w, g) instead of the three of Horner's rule; the factor 1.875 is folded into the
// tile's scaled copy: prep_tiles stores c_j = (1.875 m_j)^(-1/2), so s dX = c_j^-2 (x_j - x_i) / (1.875 r^3)
// = m_j (x_j - x_i) / r^3 with s = (c_j r)^-3 / 1.875 as the body returns it.
// Remainder 2.19 e^3 < 3e-18 per pair; measured max relative error of s 9.5e-16, mean +2e-18.
// Why not cheaper: a linear-only correction leaves 1.875 e^2 ~ 1e-12 per pair whose pair-to-pair
// fluctuation is amplified by the cancellation in the net force (the bar is the MAX over particles,
// and the unluckiest of 1e6 particles has a net force ~100x below its largest pair terms).
//
// Instruction ORDER matters on this pipe (micro-benchmarked on B200): a DFMA
// whose three source operands are three different registers that all have to come from the register
// file occupies the FP64 pipe for 3 clk instead of 2; an operand that the PREVIOUS FP64 instruction of
// the warp held in the same operand slot (SASS `.reuse`) is not read again.  So the body is written in
// stages over the R_I register-blocked i-particles of ONE source j -- all differences (they share c_j
// and X_j/Y_j/Z_j), then the <= 2-register r2 / polynomial instructions, then the accumulate triples
// (they share s) -- and the stages are separated by never-taken branches on bits of the kernel argument
// `zero`, because ptxas otherwise interleaves the stages to hide latency and loses the operand reuse
// (89-90 % instead of 84 % FP64-pipe occupancy).  Latency is hidden by the other 3 warps of the SMSP.
//
// What the scaling costs: X_j = fl(c_j x_j) carries one rounding, 1.1e-16 |x_j| / r relative to
// dX -- a few 1e-15 for the closest far pairs of these sets, random in sign (measured in the
// parity tests).
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

// Softened branches of Eq. 4 as g = calF / r in fp64.  Caller guarantees 0 < r2 < h^2.
__device__ __noinline__ double spline_g_soft_f64(double r2, double h)
{
    const double r = sqrt(r2);
    const double ih = 1.0 / h, u = r * ih, ih3 = ih * ih * ih;
    if (u < 0.5) return ih3 * (32.0 / 3.0 + u * u * (32.0 * u - 38.4));
    return ih3 * (64.0 / 3.0 + u * (-48.0 + u * (38.4 - (32.0 / 3.0) * u))) - 1.0 / (15.0 * r * r2);
}

// Integer triplets n with n.n <= 12: a superset of every n with |d - nL| < 2.6 L for |d_c| <= L/2 (Eq. 5 cut).
// Entry 0 is (0, 0, 0), the leading image.
constexpr int EWALD_NTRIPLETS = 179;
struct EwaldTriplets {
    double3 v[EWALD_NTRIPLETS];
    constexpr EwaldTriplets() : v{}
    {
        int c = 1;
        for (int a = -3; a <= 3; ++a)
            for (int b = -3; b <= 3; ++b)
                for (int d = -3; d <= 3; ++d)
                    if (a * a + b * b + d * d <= 12 && (a != 0 || b != 0 || d != 0)) { v[c].x = a; v[c].y = b; v[c].z = d; ++c; }
    }
};
__constant__ double3 ewald_triplets[EWALD_NTRIPLETS];

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

    // r2^(-3/2), 6 FP64-pipe instructions, relative error a few ulp (near body; the far body inlines the 5-op form).
    static __device__ __forceinline__ double rcube(double r2)
    {
        const double y0 = rsqrt_seed(r2);
        const double y2 = y0 * y0;
        const double e = fma(-r2, y2, 1.0);
        const double q3 = y0 * y2;
        const double t = q3 * e;
        const double p = fma(1.875, e, 1.5);
        return fma(t, p, q3);
    }

    // Running sums of the far tiles, kept in registers ACROSS tiles: the persistent driver adds them to the double-double
    // accumulator only every FAR_TILES_PER_FLUSH far tiles (and before a near tile / at the end of the i-block), so
    // the far loop of the next tile starts without waiting for the last DFMAs of this one to drain.
    struct FarSums {
        double ax[R_I], ay[R_I], az[R_I];
    };
    static constexpr int FAR_TILES_PER_FLUSH = STEPS_FP64_FAR_TILES_PER_FLUSH;
    static constexpr int FAR_SOURCES_PER_FLUSH = FAR_TILES_PER_FLUSH * TJ;      // the same, for drivers that sum parts of tiles
    static __device__ __forceinline__ void far_zero(FarSums& F)
    {
#pragma unroll
        for (int k = 0; k < R_I; ++k) F.ax[k] = F.ay[k] = F.az[k] = 0.0;
    }
    static __device__ __forceinline__ void far_flush(FarSums& F, double* acc)
    {
#pragma unroll
        for (int k = 0; k < R_I; ++k) { flush(acc, 0, k, F.ax[k]); flush(acc, 1, k, F.ay[k]); flush(acc, 2, k, F.az[k]); }
        far_zero(F);
    }

    static __device__ __forceinline__ void fold_flush(FarSums& F, double* acc) { far_flush(F, acc); }   // far_fold() sums into F like far()

    // [j0, j1): the sources of the tile to sum (the whole tile in the ring driver; a part of it in the split-j driver).
    // PREFETCH (tile record in GLOBAL memory, split-j driver): the next source is loaded one pass ahead, so that its L2
    // latency is behind the arithmetic of this pass (in shared memory the load is cheap and the registers are worth more).
    template <bool PREFETCH = false>
    static __device__ __forceinline__ void far(const Tile& T, const IState& S, FarSums& F, int zero, int j0 = 0, int j1 = TJ)
    {
        constexpr double A = 1.4;
        constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);   // (u - A)^2 + C0 = 1/1.875 at u = 1
        double (&ax)[R_I] = F.ax, (&ay)[R_I] = F.ay, (&az)[R_I] = F.az;
        double2 nXY, nZC;
        if (PREFETCH) { nXY = *reinterpret_cast<const double2*>(&T.far[j0].X); nZC = *reinterpret_cast<const double2*>(&T.far[j0].Z); }
#pragma unroll 1
        for (int j = j0; j < j1; ++j) {
            double2 XY, ZC;
            if (PREFETCH) {
                XY = nXY; ZC = nZC;
                const int jn = min(j + 1, j1 - 1);
                nXY = *reinterpret_cast<const double2*>(&T.far[jn].X); nZC = *reinterpret_cast<const double2*>(&T.far[jn].Z);
            } else {
                XY = *reinterpret_cast<const double2*>(&T.far[j].X); ZC = *reinterpret_cast<const double2*>(&T.far[j].Z);
            }
            const double X = XY.x, Y = XY.y, Z = ZC.x, C = ZC.y;
            double dX[R_I], dY[R_I], dZ[R_I], r2[R_I], y0[R_I], y2[R_I], w[R_I];
            STEPS_STAGE_FENCE(zero, 0);
#pragma unroll
            for (int k = 0; k < R_I; ++k) dX[k] = fma(-S.x[k], C, X);
#pragma unroll
            for (int k = 0; k < R_I; ++k) dY[k] = fma(-S.y[k], C, Y);
#pragma unroll
            for (int k = 0; k < R_I; ++k) dZ[k] = fma(-S.z[k], C, Z);
            STEPS_STAGE_FENCE(zero, 1);
#pragma unroll
            for (int k = 0; k < R_I; ++k) r2[k] = fma(dZ[k], dZ[k], fma(dY[k], dY[k], dX[k] * dX[k]));
#pragma unroll
            for (int k = 0; k < R_I; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                y2[k] = y0[k] * y0[k];
                w[k] = fma(r2[k], y2[k], -A);
                y2[k] = y0[k] * y2[k];
                w[k] = fma(w[k], w[k], C0);
                w[k] = y2[k] * w[k];
            }
            STEPS_STAGE_FENCE(zero, 2);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                ax[k] = fma(dX[k], w[k], ax[k]); ay[k] = fma(dY[k], w[k], ay[k]); az[k] = fma(dZ[k], w[k], az[k]);
            }
        }
    }

    // Far body in a periodic box (Eq. 5, leading image) for a (group, unit) pair that cannot be softened (box_shift in
    // common.cuh).  The image shift is already on the i-particles (`shifted`), so the pair arithmetic is the body of far()
    // plus, for the components in MASK -- those whose separations straddle half the box -- the fold d' = e - copysign(L/2, e)
    // in scaled units (h = c_j L/2, one DMUL per source): 14 + popcount(MASK) FP64-pipe instructions per interaction.
    static __device__ __forceinline__ IState shifted(const IState& S, const double (&s)[3])
    {
        IState Q;
#pragma unroll
        for (int k = 0; k < R_I; ++k) { Q.x[k] = S.x[k] + s[0]; Q.y[k] = S.y[k] + s[1]; Q.z[k] = S.z[k] + s[2]; Q.h[k] = S.h[k]; }
        return Q;
    }
    template <int MASK>
    static __device__ __forceinline__ void far_fold(const Tile& T, const IState& S, FarSums& F, int zero, double halfL,
                                                    int j0 = 0, int j1 = TJ)
    {
        constexpr double A = 1.4;
        constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);
        double (&ax)[R_I] = F.ax, (&ay)[R_I] = F.ay, (&az)[R_I] = F.az;
#pragma unroll 1
        for (int j = j0; j < j1; ++j) {
            const double2 XY = *reinterpret_cast<const double2*>(&T.far[j].X);
            const double2 ZC = *reinterpret_cast<const double2*>(&T.far[j].Z);
            const double X = XY.x, Y = XY.y, Z = ZC.x, C = ZC.y;
            const double hc = C * halfL;
            double dX[R_I], dY[R_I], dZ[R_I], r2[R_I], y0[R_I], y2[R_I], w[R_I];
            STEPS_STAGE_FENCE(zero, 0);
#pragma unroll
            for (int k = 0; k < R_I; ++k) dX[k] = fma(-S.x[k], C, X);
#pragma unroll
            for (int k = 0; k < R_I; ++k) dY[k] = fma(-S.y[k], C, Y);
#pragma unroll
            for (int k = 0; k < R_I; ++k) dZ[k] = fma(-S.z[k], C, Z);
            if (MASK & 1) {
#pragma unroll
                for (int k = 0; k < R_I; ++k) dX[k] = fold_f64(dX[k], hc);
            }
            if (MASK & 2) {
#pragma unroll
                for (int k = 0; k < R_I; ++k) dY[k] = fold_f64(dY[k], hc);
            }
            if (MASK & 4) {
#pragma unroll
                for (int k = 0; k < R_I; ++k) dZ[k] = fold_f64(dZ[k], hc);
            }
            STEPS_STAGE_FENCE(zero, 1);
#pragma unroll
            for (int k = 0; k < R_I; ++k) r2[k] = fma(dZ[k], dZ[k], fma(dY[k], dY[k], dX[k] * dX[k]));
#pragma unroll
            for (int k = 0; k < R_I; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                y2[k] = y0[k] * y0[k];
                w[k] = fma(r2[k], y2[k], -A);
                y2[k] = y0[k] * y2[k];
                w[k] = fma(w[k], w[k], C0);
                w[k] = y2[k] * w[k];
            }
            STEPS_STAGE_FENCE(zero, 2);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                ax[k] = fma(dX[k], w[k], ax[k]); ay[k] = fma(dY[k], w[k], ay[k]); az[k] = fma(dZ[k], w[k], az[k]);
            }
        }
    }

    // Leading periodic image of a separation component (Eq. 5, quasi-periodic boundary): d - L rint(d/L)
    // with the round-to-nearest-even shift trick (valid for |d/L| < 2^51), 3 FP64 instructions, no conversion.
    static __device__ __forceinline__ double wrap(double d, double L, double invL)
    {
        constexpr double SHIFT = 6755399441055744.0;                 // 1.5 * 2^52
        const double n = __dadd_rn(__fma_rn(d, invL, SHIFT), -SHIFT);
        return __fma_rn(-L, n, d);
    }

    static __device__ __forceinline__ void near(const Tile& T, const IState& S, double* acc, int j0 = 0, int j1 = TJ)
    {
        near_box<false>(T, S, acc, 0.0, 0.0, j0, j1);
    }

    // Periodic image sum, Eq. 5 (L65-70) with the paper's cut: every image x - nL of the separation with
    // |x - nL| < 2.6 L contributes through the pair law.  Around the nearest image (|d_c| <= L/2) these are among the
    // triplets with |n| < 2.6 + sqrt(3)/2, i.e. n.n <= 12: 179 of them; `tab` holds their offsets n L (3 doubles each,
    // entry 0 = the nearest image) in shared memory.  Every image other than the nearest is at least L/2 away, so when
    // h_i + h_j <= L/2 (any sane softening) only the nearest image can be softened: it goes through the near body
    // (spline test), the other 178 through a branch-free Newtonian body -- 3 DADD, 3 for r^2, the 5-instruction r^-3 of
    // the far body, 3 DFMA = 14 FP64-pipe instructions per image -- with the cut applied as an integer compare of the
    // bit patterns (ALU pipe, not FP64) and m_j multiplied once per pair.  Pairs with h_i + h_j > L/2 take the general loop.
    static __device__ __forceinline__ void near_images(const Tile& T, const IState& S, double* acc, double L, double invL,
                                                       const double* __restrict__ tab, int j0 = 0, int j1 = TJ)
    {
        near_images_view(T.x, T.y, T.z, T.m, T.h, S, acc, L, invL, tab, j0, j1);
    }
    // The same on any copy of the plain sources (x, y, z, m, h), e.g. one staged in shared memory.
    static __device__ __forceinline__ void near_images_view(const double* __restrict__ Tx, const double* __restrict__ Ty,
                                                            const double* __restrict__ Tz, const double* __restrict__ Tm,
                                                            const double* __restrict__ Th, const IState& S, double* acc, double L,
                                                            double invL, const double* __restrict__ tab, int j0, int j1)
    {
        constexpr double A = 1.4;
        constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);
        const double cut2 = (2.6 * L) * (2.6 * L), halfL = 0.5 * L;
        const long long cut2_bits = __double_as_longlong(cut2);
#pragma unroll 1
        for (int j = j0; j < j1; ++j) {
            const double xj = Tx[j], yj = Ty[j], zj = Tz[j], mq = Tm[j], hj = Th[j];
            if (mq == 0.0) continue;                                   // pads and massless sources (warp-uniform)
            // px: sum over the images of s v, in units of 1 / STEPS_FP64_FOLD (the far body's r^-3 carries that factor)
            double dx[R_I], dy[R_I], dz[R_I], px[R_I], py[R_I], pz[R_I];
            bool newtonian = true;
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                dx[k] = wrap(xj - S.x[k], L, invL); dy[k] = wrap(yj - S.y[k], L, invL); dz[k] = wrap(zj - S.z[k], L, invL);
                const double hs = S.h[k] + hj;
                newtonian = newtonian && hs <= halfL;
                const double r2 = fma(dz[k], dz[k], fma(dy[k], dy[k], dx[k] * dx[k]));
                double s0 = rcube(r2);                                // the nearest image: Eq. 4 in full (readings #2, #4)
                if (r2 < hs * hs || r2 == 0.0) s0 = (r2 == 0.0) ? 0.0 : spline_g_soft_f64(r2, hs);
                s0 *= 1.0 / STEPS_FP64_FOLD;
                px[k] = dx[k] * s0; py[k] = dy[k] * s0; pz[k] = dz[k] * s0;
            }
            if (__all_sync(0xffffffffu, newtonian)) {
                // the 178 other triplets, for two of the thread's particles at a time (as in far_images: all four at once
                // exceed the registers and their dependent chains run one after the other)
                constexpr int H = 2;
                static_assert(R_I % H == 0, "whole passes");
#pragma unroll
                for (int k0 = 0; k0 < R_I; k0 += H) {
#pragma unroll 2
                    for (int c = 1; c < EWALD_NTRIPLETS; ++c) {
                        const double ox = tab[3 * c], oy = tab[3 * c + 1], oz = tab[3 * c + 2];
                        double vx[H], vy[H], vz[H], r2[H], y0[H], y2[H], w[H];
#pragma unroll
                        for (int k = 0; k < H; ++k) { vx[k] = dx[k0 + k] - ox; vy[k] = dy[k0 + k] - oy; vz[k] = dz[k0 + k] - oz; }
#pragma unroll
                        for (int k = 0; k < H; ++k) r2[k] = fma(vz[k], vz[k], fma(vy[k], vy[k], vx[k] * vx[k]));
#pragma unroll
                        for (int k = 0; k < H; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
                        for (int k = 0; k < H; ++k) {
                            y2[k] = y0[k] * y0[k];
                            w[k] = fma(r2[k], y2[k], -A);
                            y2[k] = y0[k] * y2[k];
                            w[k] = fma(w[k], w[k], C0);
                            w[k] = y2[k] * w[k];
                            if (!(__double_as_longlong(r2[k]) < cut2_bits)) w[k] = 0.0;   // "|x - nL| < 2.6 L", strict (r2 >= 0)
                        }
#pragma unroll
                        for (int k = 0; k < H; ++k) {
                            px[k0 + k] = fma(vx[k], w[k], px[k0 + k]); py[k0 + k] = fma(vy[k], w[k], py[k0 + k]);
                            pz[k0 + k] = fma(vz[k], w[k], pz[k0 + k]);
                        }
                    }
                }
            } else {                                                   // some h_i + h_j > L/2: every image through Eq. 4
#pragma unroll 1
                for (int c = 1; c < EWALD_NTRIPLETS; ++c) {
                    const double ox = tab[3 * c], oy = tab[3 * c + 1], oz = tab[3 * c + 2];
#pragma unroll
                    for (int k = 0; k < R_I; ++k) {
                        const double vx = dx[k] - ox, vy = dy[k] - oy, vz = dz[k] - oz;
                        const double r2 = fma(vz, vz, fma(vy, vy, vx * vx));
                        const double hs = S.h[k] + hj;
                        double s = rcube(r2);
                        if (r2 < hs * hs) s = spline_g_soft_f64(r2, hs);
                        if (!(r2 < cut2)) s = 0.0;
                        s *= 1.0 / STEPS_FP64_FOLD;
                        px[k] = fma(vx, s, px[k]); py[k] = fma(vy, s, py[k]); pz[k] = fma(vz, s, pz[k]);
                    }
                }
            }
            const double mf = STEPS_FP64_FOLD * mq;
#pragma unroll
            for (int k = 0; k < R_I; ++k) { flush(acc, 0, k, mf * px[k]); flush(acc, 1, k, mf * py[k]); flush(acc, 2, k, mf * pz[k]); }
        }
    }

    // The image sum for a (group, tile) pair NO image of which can be softened (the driver's box test), with the candidate
    // images pruned from the two bounding boxes: `Q` carries the pair's common lattice shift (so every separation
    // d = x_j - x_i' lies in the box-difference interval the driver pruned against -- no per-pair wrap: the image SET
    // {d - nL : |d - nL| < 2.6 L} does not depend on the representative, reading #17), `cand[0..ncand)` are the indices
    // into `tab` (offsets n L, n in [-3, 3]^3) of the images that come within the cut for SOME pair of the two boxes --
    // about 90 for compact cells instead of the 179 a single pair needs in the worst case.  Every image runs the
    // branch-free 14-instruction Newtonian body, the cut as an integer compare.
    // (Tx, Ty, Tz, Tm: the tile's plain sources, e.g. staged in shared memory; [j0, j1): the sources to sum.)
    // The candidates are walked twice per source, for two of the thread's four particles at a time: with all four in one
    // pass the live values (separations, sums, temporaries) exceed the register file and ptxas runs the four dependent
    // 12-instruction chains one after the other (FP64 pipe 66 % active, measured); two at a time they interleave.
    static __device__ __forceinline__ void far_images(const double* __restrict__ Tx, const double* __restrict__ Ty,
                                                      const double* __restrict__ Tz, const double* __restrict__ Tm, const IState& Q,
                                                      double* acc, double L, const double* __restrict__ tab,
                                                      const unsigned short* __restrict__ cand, int ncand, int j0, int j1)
    {
        constexpr double A = 1.4;
        constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);
        constexpr int H = 2;                                           // particles per pass
        static_assert(R_I % H == 0, "whole passes");
        const long long cut2_bits = __double_as_longlong((2.6 * L) * (2.6 * L));
        if (ncand <= 0) return;                                        // (only a slice of pads has no candidate)
#pragma unroll 1
        for (int j = j0; j < j1; ++j) {
            const double xj = Tx[j], yj = Ty[j], zj = Tz[j], mq = Tm[j];
            if (mq == 0.0) continue;                                   // pads and massless sources (warp-uniform)
            const double mf = STEPS_FP64_FOLD * mq;
#pragma unroll
            for (int k0 = 0; k0 < R_I; k0 += H) {
                double dx[H], dy[H], dz[H], px[H], py[H], pz[H];
#pragma unroll
                for (int k = 0; k < H; ++k) {
                    dx[k] = xj - Q.x[k0 + k]; dy[k] = yj - Q.y[k0 + k]; dz[k] = zj - Q.z[k0 + k];
                    px[k] = py[k] = pz[k] = 0.0;
                }
                // (the next candidate's offsets are fetched one pass ahead: index -> address -> three loads is a dependent
                // chain of two shared-memory latencies that would otherwise open every pass)
                double nox, noy, noz;
                { const int t3 = 3 * cand[0]; nox = tab[t3]; noy = tab[t3 + 1]; noz = tab[t3 + 2]; }
#pragma unroll 2
                for (int c = 0; c < ncand; ++c) {
                    const double ox = nox, oy = noy, oz = noz;
                    { const int t3 = 3 * cand[min(c + 1, ncand - 1)]; nox = tab[t3]; noy = tab[t3 + 1]; noz = tab[t3 + 2]; }
                    double vx[H], vy[H], vz[H], r2[H], y0[H], y2[H], w[H];
#pragma unroll
                    for (int k = 0; k < H; ++k) { vx[k] = dx[k] - ox; vy[k] = dy[k] - oy; vz[k] = dz[k] - oz; }
#pragma unroll
                    for (int k = 0; k < H; ++k) r2[k] = fma(vz[k], vz[k], fma(vy[k], vy[k], vx[k] * vx[k]));
#pragma unroll
                    for (int k = 0; k < H; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
                    for (int k = 0; k < H; ++k) {
                        y2[k] = y0[k] * y0[k];
                        w[k] = fma(r2[k], y2[k], -A);
                        y2[k] = y0[k] * y2[k];
                        w[k] = fma(w[k], w[k], C0);
                        w[k] = y2[k] * w[k];
                        if (!(__double_as_longlong(r2[k]) < cut2_bits)) w[k] = 0.0;   // "|x - nL| < 2.6 L", strict (r2 >= 0)
                    }
#pragma unroll
                    for (int k = 0; k < H; ++k) {
                        px[k] = fma(vx[k], w[k], px[k]); py[k] = fma(vy[k], w[k], py[k]); pz[k] = fma(vz[k], w[k], pz[k]);
                    }
                }
#pragma unroll
                for (int k = 0; k < H; ++k) { flush(acc, 0, k0 + k, mf * px[k]); flush(acc, 1, k0 + k, mf * py[k]); flush(acc, 2, k0 + k, mf * pz[k]); }
            }
        }
    }

    // PERIODIC: every separation is replaced by its leading image in a cubic box of side L (row 8(f)-3).
    template <bool PERIODIC>
    static __device__ __forceinline__ void near_box(const Tile& T, const IState& S, double* acc, double L, double invL,
                                                    int j0 = 0, int j1 = TJ)
    {
        near_view<PERIODIC>(T.x, T.y, T.z, T.m, T.h, S, acc, L, invL, j0, j1);
    }
    // One source against the thread's R_I particles through all three branches of Eq. 4.
    template <bool PERIODIC>
    static __device__ __forceinline__ void near_one(double xj, double yj, double zj, double mq, double hj, const IState& S,
                                                    double (&ax)[R_I], double (&ay)[R_I], double (&az)[R_I], double L, double invL)
    {
#pragma unroll
        for (int k = 0; k < R_I; ++k) {
            double dx = xj - S.x[k], dy = yj - S.y[k], dz = zj - S.z[k];
            if (PERIODIC) { dx = wrap(dx, L, invL); dy = wrap(dy, L, invL); dz = wrap(dz, L, invL); }
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double hs = S.h[k] + hj;
            double s = mq * rcube(r2);
            if (r2 < hs * hs || r2 == 0.0)                        // Eq. 4 branches 1-2; readings #2, #4
                s = (r2 == 0.0) ? 0.0 : mq * spline_g_soft_f64(r2, hs);
            ax[k] = fma(dx, s, ax[k]); ay[k] = fma(dy, s, ay[k]); az[k] = fma(dz, s, az[k]);
        }
    }
    // The same on any copy of the plain sources (x, y, z, m, h), e.g. one staged in shared memory.
    template <bool PERIODIC>
    static __device__ __forceinline__ void near_view(const double* __restrict__ Tx, const double* __restrict__ Ty,
                                                     const double* __restrict__ Tz, const double* __restrict__ Tm,
                                                     const double* __restrict__ Th, const IState& S, double* acc, double L,
                                                     double invL, int j0, int j1)
    {
        double ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) ax[k] = ay[k] = az[k] = 0.0;
#pragma unroll 1
        for (int j = j0; j < j1; ++j) near_one<PERIODIC>(Tx[j], Ty[j], Tz[j], Tm[j], Th[j], S, ax, ay, az, L, invL);
#pragma unroll
        for (int k = 0; k < R_I; ++k) { flush(acc, 0, k, ax[k]); flush(acc, 1, k, ay[k]); flush(acc, 2, k, az[k]); }
    }
    // The same for a tile record in GLOBAL memory (the group-ring driver's general tiles): a warp-uniform load per source
    // would pay the L2 latency at every source; instead every lane loads one source of 32 (coalesced) and the warp hands
    // them round by shuffle.  [j0, j1) must be whole sets of 32.
    template <bool PERIODIC>
    static __device__ __forceinline__ void near_global(const Tile& T, const IState& S, double* acc, double L, double invL, int j0, int j1)
    {
        const int lane = threadIdx.x & 31;
        double ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) ax[k] = ay[k] = az[k] = 0.0;
#pragma unroll 1
        for (int jb = j0; jb < j1; jb += 32) {
            const double lx = T.x[jb + lane], ly = T.y[jb + lane], lz = T.z[jb + lane], lm = T.m[jb + lane], lh = T.h[jb + lane];
#pragma unroll 1
            for (int s = 0; s < 32; ++s)
                near_one<PERIODIC>(__shfl_sync(0xffffffffu, lx, s), __shfl_sync(0xffffffffu, ly, s), __shfl_sync(0xffffffffu, lz, s),
                                   __shfl_sync(0xffffffffu, lm, s), __shfl_sync(0xffffffffu, lh, s), S, ax, ay, az, L, invL);
        }
#pragma unroll
        for (int k = 0; k < R_I; ++k) { flush(acc, 0, k, ax[k]); flush(acc, 1, k, ay[k]); flush(acc, 2, k, az[k]); }
    }
};

}  // namespace steps
