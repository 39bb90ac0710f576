// kdk.cuh -- rows a4/a5/a7: fused kick/drift pass (Eq. 9-10, applied to
// Eq. 8) and the momentum diagnostic.  HBM-bound: 5 doubles in/out per component.
#pragma once
#include "common.cuh"

namespace steps {

struct KdkScalars {
    double ac, bc, ao, bo, gamma, B;
};

// Elementwise over the 3N components (SoA makes x/v/acc component k line up).
__global__ void __launch_bounds__(256) kick_drift_kernel(double* __restrict__ pos, double* __restrict__ vel,
                                                         const double* __restrict__ acc, long long M, KdkScalars c)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < M; k += stride) {
        const double x = pos[k];
        const double g = fma(c.B, x, acc[k]);          // acc + B x  (background term, reading #6)
        double v = vel[k];
        v = fma(c.bc, g, c.ac * v);                     // closing half kick of the previous step
        v = fma(c.bo, g, c.ao * v);                     // opening half kick of this step
        vel[k] = v;
        pos[k] = fma(c.gamma, v, x);                    // drift
    }
}

constexpr int MOM_BLOCKS = 148;

// Stage 1: fixed assignment of particles to blocks/threads, fixed-order tree -> deterministic.
__global__ void __launch_bounds__(256) momentum_stage1(const double* __restrict__ vec, const double* __restrict__ mass,
                                                        long long N, double* __restrict__ partial)
{
    double s[4] = {0, 0, 0, 0};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
        const double m = mass[i], vx = vec[i], vy = vec[N + i], vz = vec[2 * N + i];
        s[0] = fma(m, vx, s[0]); s[1] = fma(m, vy, s[1]); s[2] = fma(m, vz, s[2]);
        s[3] = fma(m, sqrt(vx * vx + vy * vy + vz * vz), s[3]);
    }
    __shared__ double sh[8][4];
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_down_sync(0xffffffffu, s[c], o);
    if ((threadIdx.x & 31) == 0)
        for (int c = 0; c < 4; ++c) sh[threadIdx.x >> 5][c] = s[c];
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0;
        for (int w = 0; w < 8; ++w) t += sh[w][threadIdx.x];
        partial[blockIdx.x * 4 + threadIdx.x] = t;
    }
}

__global__ void momentum_stage2(const double* __restrict__ partial, int nblocks, double* __restrict__ out4)
{
    if (threadIdx.x < 4) {
        double t = 0;
        for (int b = 0; b < nblocks; ++b) t += partial[b * 4 + threadIdx.x];
        out4[threadIdx.x] = t;
    }
}

// ---- adaptive global time step, Eq. 12 (L113-116) ---------------------------------------------------------
// dt = min[dt_max, min_i sqrt(2 eta_i eps / |A_i|)], eta_i = 2.8 h_i, A_i = coef (acc_i + B x_i) (reading #11).
// Each particle's candidate is formed exactly as the formula reads (IEEE fp64 sqrt and divide); the minimum is exact, so
// the result does not depend on the reduction order.  |A_i| = 0 puts no limit.  48 B read per particle, HBM/L2-bound.
__global__ void __launch_bounds__(256) timestep_stage1(const double* __restrict__ pos, const double* __restrict__ acc,
                                                        const double* __restrict__ soft, long long N, double coef, double B,
                                                        double eps, double dt_max, double* __restrict__ partial)
{
    double dt = dt_max;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride)
        dt = eq12_candidate(acc[i], acc[N + i], acc[2 * N + i], pos[i], pos[N + i], pos[2 * N + i], soft[i], coef, B, eps, dt);
    __shared__ double sh[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dt = fmin(dt, __shfl_down_sync(0xffffffffu, dt, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = dt;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) dt = fmin(dt, sh[w]);
        partial[blockIdx.x] = dt;
    }
}

__global__ void timestep_stage2(const double* __restrict__ partial, int nblocks, double* __restrict__ out)
{
    if (threadIdx.x == 0) {
        double dt = partial[0];
        for (int b = 1; b < nblocks; ++b) dt = fmin(dt, partial[b]);
        out[0] = dt;
    }
}

// ---- net-force residual, the convergence monitor of glass generation (section 3.1) --------------
// g_i = acc_i + B x_i;  out = {sum_i |g_i|^2, max_i |g_i|}.  Fixed assignment + fixed-order tree: deterministic.
__global__ void __launch_bounds__(256) residual_stage1(const double* __restrict__ pos, const double* __restrict__ acc,
                                                        long long N, double B, double* __restrict__ partial)
{
    double s = 0.0, mx = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
        const double gx = fma(B, pos[i], acc[i]), gy = fma(B, pos[N + i], acc[N + i]), gz = fma(B, pos[2 * N + i], acc[2 * N + i]);
        const double g2 = fma(gz, gz, fma(gy, gy, gx * gx));
        s += g2;
        mx = fmax(mx, sqrt(g2));
    }
    __shared__ double sh[8][2];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s += __shfl_down_sync(0xffffffffu, s, o);
        mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][0] = s; sh[threadIdx.x >> 5][1] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { s += sh[w][0]; mx = fmax(mx, sh[w][1]); }
        partial[2 * blockIdx.x] = s; partial[2 * blockIdx.x + 1] = mx;
    }
}

__global__ void residual_stage2(const double* __restrict__ partial, int nblocks, double* __restrict__ out2)
{
    if (threadIdx.x == 0) {
        double s = 0.0, mx = 0.0;
        for (int b = 0; b < nblocks; ++b) { s += partial[2 * b]; mx = fmax(mx, partial[2 * b + 1]); }
        out2[0] = s; out2[1] = mx;
    }
}

// ---- device-resident adaptive stepping (second half): no host round trip between steps -----------
// Run state in device memory: {a, dt, alpha_close, beta_close, steps taken}.
struct RunState {
    double a, dt, alpha_close, beta_close, steps;
};
struct CosmoScalars {
    double H0, Om, Or, OL, Ok;
};
__device__ __forceinline__ double hubble_dev(double a, const CosmoScalars& c)          // PAPER.md Eq. 1 (L37)
{
    return c.H0 * sqrt(c.Om / (a * a * a) + c.Or / (a * a * a * a) + c.OL + c.Ok / (a * a));
}

// Eq. 12 with coef = |G| a^-3 taken from the run state (stage 1 of the two-stage exact minimum).
__global__ void __launch_bounds__(256) timestep_state_stage1(const double* __restrict__ pos, const double* __restrict__ acc,
                                                              const double* __restrict__ soft, long long N,
                                                              const RunState* __restrict__ st, double absG, double B,
                                                              double eps, double dt_max, double* __restrict__ partial)
{
    const double a = st->a;
    const double coef = absG / (a * a * a);
    double dt = dt_max;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride)
        dt = eq12_candidate(acc[i], acc[N + i], acc[2 * N + i], pos[i], pos[N + i], pos[2 * N + i], soft[i], coef, B, eps, dt);
    __shared__ double sh[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dt = fmin(dt, __shfl_down_sync(0xffffffffu, dt, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = dt;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) dt = fmin(dt, sh[w]);
        partial[blockIdx.x] = dt;
    }
}

// Stage 2 + the step's coefficients (the arithmetic of steps_kdk_schedule, on the device): writes the six kick/drift
// scalars of THIS step to coef6 = {alpha_close(prev), beta_close(prev), alpha_open, beta_open, gamma, B} and advances
// the state to a_{n+1} with the new closing coefficients.
// fused_bits != nullptr: the minimum over the particles was folded into *fused_bits by the previous force evaluation
// (Eq12Fuse in common.cuh) instead of into `partial` (all bits set = no particle put a limit: NaN, which fmin ignores).
__global__ void step_coefficients_kernel(const double* __restrict__ partial, int nblocks, RunState* __restrict__ st,
                                         CosmoScalars c, double G, double B, double* __restrict__ coef6,
                                         unsigned long long* __restrict__ fused_bits, double dt_max)
{
    if (threadIdx.x != 0) return;
    double dt;
    if (fused_bits != nullptr) {
        dt = fmin(dt_max, __longlong_as_double((long long)*fused_bits));
    } else {
        dt = partial[0];
        for (int b = 1; b < nblocks; ++b) dt = fmin(dt, partial[b]);
    }
    const double a_n = st->a;
    const bool is_static = (c.H0 == 0.0);
    const double H_n = is_static ? 0.0 : hubble_dev(a_n, c);
    double a_1 = a_n;
    if (!is_static) {                                                   // classical RK4 on da/dt = a H(a) (L127)
        const double k1 = a_n * hubble_dev(a_n, c);
        const double s2 = a_n + 0.5 * dt * k1, k2 = s2 * hubble_dev(s2, c);
        const double s3 = a_n + 0.5 * dt * k2, k3 = s3 * hubble_dev(s3, c);
        const double s4 = a_n + dt * k3, k4 = s4 * hubble_dev(s4, c);
        a_1 = a_n + dt / 6.0 * (k1 + 2.0 * (k2 + k3) + k4);
    }
    const double H_1 = is_static ? 0.0 : hubble_dev(a_1, c);
    coef6[0] = st->alpha_close; coef6[1] = st->beta_close;
    coef6[2] = 1.0 - H_n * dt;
    coef6[3] = 0.5 * dt * G / (a_n * a_n * a_n);
    coef6[4] = dt;
    coef6[5] = B;
    const double ac = 1.0 / (1.0 + H_1 * dt);
    st->alpha_close = ac;
    st->beta_close = 0.5 * dt * G / (a_1 * a_1 * a_1) * ac;
    st->a = a_1;
    st->dt = dt;
    st->steps += 1.0;
}

// The final closing half kick of a run: coefficients from the state, which is reset to the identity.
__global__ void close_coefficients_kernel(RunState* __restrict__ st, double B, double* __restrict__ coef6)
{
    if (threadIdx.x != 0) return;
    coef6[0] = st->alpha_close; coef6[1] = st->beta_close; coef6[2] = 1.0; coef6[3] = 0.0; coef6[4] = 0.0; coef6[5] = B;
    st->alpha_close = 1.0; st->beta_close = 0.0;
}

// kick_drift_kernel with its six scalars read from device memory.
__global__ void __launch_bounds__(256) kick_drift_dev_kernel(double* __restrict__ pos, double* __restrict__ vel,
                                                             const double* __restrict__ acc, long long M,
                                                             const double* __restrict__ coef6)
{
    const double ac = coef6[0], bc = coef6[1], ao = coef6[2], bo = coef6[3], gamma = coef6[4], B = coef6[5];
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < M; k += stride) {
        const double x = pos[k];
        const double g = fma(B, x, acc[k]);
        double v = vel[k];
        v = fma(bc, g, ac * v);
        v = fma(bo, g, ao * v);
        vel[k] = v;
        pos[k] = fma(gamma, v, x);
    }
}

}  // namespace steps
