// force_mixed.cuh -- pair arithmetic of the MIXED path: fp32 pairs, fp64 accumulation.
//
// Rows a1/a2 of the hot path (Eq. 8 L88 first term; Eq. 3-4):
//   far  tile: acc_i += m_j (x_j - x_i) / r^3                 (calF = 1/r^2 for r >= h, Eq. 4 third case)
//   near tile: acc_i += m_j g(r, h_i + h_j) (x_j - x_i)       (all three branches; j = i and r = 0 add 0)
//
// Far body: two j-particles per instruction with the sm_100a packed fp32x2 pipe ops
// (FADD2/FMUL2/FFMA2): 12 packed FP32-pipe instructions + 2 MUFU.RSQ per TWO interactions,
// i.e. 12 FP32-lane-cycles and 7 issue slots per interaction.  j-data is read from the
// shared-memory tile with broadcast LDS.128 (4 j per load per component), amortised over
// R_I = 4 register-blocked i-particles per thread.  Partial sums live in fp32 for one tile
// (<= 256 terms per packed half) and are then flushed into fp64 accumulators.
#pragma once
#include "common.cuh"

namespace steps {

// Softened branches of Eq. 4 as g = calF / r, evaluated in fp64 (rare path: ~1e-4 of the pairs
// of a near tile), r^2 and h = h_i + h_j given in fp32.  Caller guarantees 0 < r^2 < h^2.
__device__ __noinline__ float spline_g_soft_from_f32(float r2, float hs)
{
    const double r = sqrt((double)r2), h = (double)hs;
    const double ih = 1.0 / h, u = r * ih, ih3 = ih * ih * ih;
    double g;
    if (u < 0.5) {
        g = ih3 * (32.0 / 3.0 + u * u * (32.0 * u - 38.4));
    } else {
        g = ih3 * (64.0 / 3.0 + u * (-48.0 + u * (38.4 - (32.0 / 3.0) * u))) - 1.0 / (15.0 * r * r * r);
    }
    return (float)g;
}

struct MixedPath {
    using Tile = TileF32;

    static constexpr int NOUT = 3;            // doubles per i-particle in the accumulator / partial record

    struct IState {
        float x[R_I], y[R_I], z[R_I], h[R_I];
    };

    // acc: this thread's fp64 accumulators in shared memory, element (c, k) at acc[(c * R_I + k) * CTA_THREADS].
    static __device__ __forceinline__ void flush(double* acc, int c, int k, float partial)
    {
        double* a = acc + (c * R_I + k) * CTA_THREADS;
        *a += (double)partial;
    }

    // Loads the thread's R_I i-particles (indices already clamped into [0, N)).
    static __device__ __forceinline__ void load_i(IState& S, const double* __restrict__ pos,
                                                  const double* __restrict__ soft, long long N,
                                                  const long long (&idx)[R_I], float& rlo, float& rhi, float& hh)
    {
#pragma unroll
        for (int k = 0; k < R_I; ++k) {
            const double x = pos[idx[k]], y = pos[N + idx[k]], z = pos[2 * N + idx[k]], h = soft[idx[k]];
            S.x[k] = (float)x; S.y[k] = (float)y; S.z[k] = (float)z; S.h[k] = (float)h;
            const double r = sqrt(x * x + y * y + z * z);
            rlo = fminf(rlo, __double2float_rd(r));
            rhi = fmaxf(rhi, __double2float_ru(r));
            hh = fmaxf(hh, __double2float_ru(h));
        }
    }

    // One packed pair-of-interactions: i against (j, j+1).
    static __device__ __forceinline__ void pair2(u64 xj, u64 yj, u64 zj, u64 mj, u64 xi, u64 yi, u64 zi,
                                                 u64& ax, u64& ay, u64& az)
    {
        const u64 dx = sub2(xj, xi), dy = sub2(yj, yi), dz = sub2(zj, zi);
        const u64 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
        float a, b;
        unpack2(r2, a, b);
        const u64 rinv = pack2(rsqrt_approx(a), rsqrt_approx(b));
        const u64 s = mul2(mul2(mj, rinv), mul2(rinv, rinv));
        ax = fma2(dx, s, ax);
        ay = fma2(dy, s, ay);
        az = fma2(dz, s, az);
    }

    static __device__ __forceinline__ void far(const Tile& T, const IState& S, double* acc)
    {
        u64 xi[R_I], yi[R_I], zi[R_I], ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) {
            xi[k] = pack2(S.x[k], S.x[k]); yi[k] = pack2(S.y[k], S.y[k]); zi[k] = pack2(S.z[k], S.z[k]);
            ax[k] = ay[k] = az[k] = 0ull;
        }
#pragma unroll 2
        for (int j = 0; j < TJ; j += 4) {
            const ulonglong2 X = *reinterpret_cast<const ulonglong2*>(&T.x[j]);
            const ulonglong2 Y = *reinterpret_cast<const ulonglong2*>(&T.y[j]);
            const ulonglong2 Z = *reinterpret_cast<const ulonglong2*>(&T.z[j]);
            const ulonglong2 M = *reinterpret_cast<const ulonglong2*>(&T.m[j]);
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                pair2(X.x, Y.x, Z.x, M.x, xi[k], yi[k], zi[k], ax[k], ay[k], az[k]);
                pair2(X.y, Y.y, Z.y, M.y, xi[k], yi[k], zi[k], ax[k], ay[k], az[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < R_I; ++k) {
            float lo, hi;
            unpack2(ax[k], lo, hi); flush(acc, 0, k, lo + hi);
            unpack2(ay[k], lo, hi); flush(acc, 1, k, lo + hi);
            unpack2(az[k], lo, hi); flush(acc, 2, k, lo + hi);
        }
    }

    static __device__ __forceinline__ void near(const Tile& T, const IState& S, double* acc)
    {
        float ax[R_I], ay[R_I], az[R_I];
#pragma unroll
        for (int k = 0; k < R_I; ++k) ax[k] = ay[k] = az[k] = 0.0f;
#pragma unroll 2
        for (int j = 0; j < TJ; ++j) {
            const float xj = T.x[j], yj = T.y[j], zj = T.z[j], mj = T.m[j], hj = T.h[j];
#pragma unroll
            for (int k = 0; k < R_I; ++k) {
                const float dx = xj - S.x[k], dy = yj - S.y[k], dz = zj - S.z[k];
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                const float hs = S.h[k] + hj;
                const float rinv = rsqrt_approx(r2);
                float s = mj * rinv * (rinv * rinv);
                if (r2 < hs * hs || r2 == 0.0f)                       // Eq. 4 branches 1-2; readings #2, #4
                    s = (r2 == 0.0f) ? 0.0f : mj * spline_g_soft_from_f32(r2, hs);
                ax[k] = fmaf(dx, s, ax[k]);
                ay[k] = fmaf(dy, s, ay[k]);
                az[k] = fmaf(dz, s, az[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < R_I; ++k) {
            flush(acc, 0, k, ax[k]); flush(acc, 1, k, ay[k]); flush(acc, 2, k, az[k]);
        }
    }
};

}  // namespace steps
