// fp64_pipe_probe.cu -- micro-benchmarks behind DESIGN.md section 6.1: how long an FP64-pipe instruction holds the
// pipe on B200 as a function of where its operands come from, what a shared-memory load costs next to a saturated
// DFMA stream, and what the 14-instruction far body of force_fp64.cuh reaches in isolation with and without stage fences.
// Not part of libsteps_b200.so (build.py compiles csrc/*.cu only).  Build and run on a B200:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o fp64_pipe_probe \
//        paper_1811_05903_b200/csrc/probe/fp64_pipe_probe.cu && ./fp64_pipe_probe
// Every kernel: one CTA of 512 threads per SM (4 warps per SM sub-partition), clock64() around the loop, the slowest SM
// counts.  "clk" = cycles per warp-instruction per sub-partition; 2.00 = the nominal 64 FP64 lanes per SM.
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cuda_runtime.h>
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at line %d\n", cudaGetErrorString(e_), __LINE__); exit(1); } } while (0)
constexpr int THREADS = 512, SMS = 148, ILP = 8;

// ---- 1. operand patterns ------------------------------------------------------------------------------------------------
// PAT 0: DMUL a = a*b0            1: DFMA a = b_i*b_i + a (2 distinct)     2: DFMA a_i = b_i*c_i + a_i (3 distinct, no reuse)
//     3: DFMA a_i = b_i*c0 + a_i  (one shared operand)                     4: DFMA a_i = a_i*b0 + c0 (two shared operands)
template <int PAT>
__global__ void __launch_bounds__(THREADS, 1) pattern_kernel(const double* in, double* out, int iters, long long* clk)
{
    double a[ILP], b[ILP], c[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { a[i] = in[threadIdx.x + i]; b[i] = in[threadIdx.x + 8 + i]; c[i] = in[threadIdx.x + 16 + i]; }
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int i = 0; i < ILP; ++i) {
                if (PAT == 0) asm volatile("mul.rn.f64 %0, %0, %1;" : "+d"(a[i]) : "d"(b[0]));
                if (PAT == 1) asm volatile("fma.rn.f64 %0, %1, %1, %0;" : "+d"(a[i]) : "d"(b[i]));
                if (PAT == 2) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(a[i]) : "d"(b[i]), "d"(c[i]));
                if (PAT == 3) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(a[i]) : "d"(b[i]), "d"(c[0]));
                if (PAT == 4) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(a[i]) : "d"(b[0]), "d"(c[0]));
            }
        }
    }
    const long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += a[i] + b[i] + c[i];
    out[blockIdx.x * THREADS + threadIdx.x] = s;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// ---- 2. shared-memory loads next to 56 two-source DFMAs per pass -------------------------------------------------------------
// MODE 0: none    1: 4 broadcast LDS.64 per pass    2: 2 broadcast LDS.128 per pass   (the loaded values feed 4 of the DFMAs)
template <int MODE>
__global__ void __launch_bounds__(THREADS, 1) lds_kernel(const double* in, double* out, int iters, long long* clk)
{
    __shared__ __align__(16) double sm[1024];
    for (int i = threadIdx.x; i < 1024; i += THREADS) sm[i] = in[i];
    __syncthreads();
    double a[ILP], b[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { a[i] = in[threadIdx.x + i]; b[i] = in[threadIdx.x + 8 + i]; }
    double l0 = 0, l1 = 0, l2 = 0, l3 = 0;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        if (MODE == 1) { const int j = it & 255; l0 = sm[j]; l1 = sm[256 + j]; l2 = sm[512 + j]; l3 = sm[768 + j]; }
        if (MODE == 2) {
            const int j = (it & 127) * 2;
            const double2 u = *reinterpret_cast<const double2*>(sm + j), v = *reinterpret_cast<const double2*>(sm + 256 + j);
            l0 = u.x; l1 = u.y; l2 = v.x; l3 = v.y;
        }
#pragma unroll
        for (int r = 0; r < 7; ++r) {
#pragma unroll
            for (int i = 0; i < ILP; ++i) {
                if (r == 0 && i < 4 && MODE >= 1) {
                    const double l = i == 0 ? l0 : i == 1 ? l1 : i == 2 ? l2 : l3;
                    asm volatile("fma.rn.f64 %0, %1, %1, %0;" : "+d"(a[i]) : "d"(l));
                } else {
                    asm volatile("fma.rn.f64 %0, %1, %1, %0;" : "+d"(a[i]) : "d"(b[i]));
                }
            }
        }
    }
    const long long t1 = clock64();
    double s = l0 + l1 + l2 + l3;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += a[i] + b[i];
    out[blockIdx.x * THREADS + threadIdx.x] = s;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// ---- 3. the 14-instruction far body in isolation ----------------------------------------------------------------------------
// ORDER 0: two sources x 4 i per pass, written interaction by interaction (ptxas schedules freely)
// ORDER 1: one source x 4 i per pass in three stages separated by never-taken branches (the body of force_fp64.cuh)
// ORDER 2: as 1, the tile walked by pointer increment: ptxas then addresses the loads through a uniform register
//          (LDS [UR]) instead of a per-lane register (LDS [R+UR]), which needs no register-file read
__device__ __forceinline__ double seed64h(double r2) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r2)); return y; }
#define FENCE(zero, n) asm volatile("{\n.reg .pred p;\n.reg .b32 t;\nand.b32 t, %0, %1;\nsetp.ne.s32 p, t, 0;\n@p trap;\n}" :: "r"(zero), "r"(1 << (n)))
template <int ORDER>
__global__ void __launch_bounds__(THREADS, 1) far_kernel(const double* __restrict__ tile, double* out, int ntiles, long long* clk, int zero)
{
    constexpr int RI = 4;
    constexpr double A = 1.4, C0 = 1.0 / 1.875 - (1.0 - A) * (1.0 - A);
    __shared__ __align__(16) double T[256][4];                   // (X, Y, Z, c) per source
    for (int i = threadIdx.x; i < 1024; i += THREADS) (&T[0][0])[i] = tile[i];
    __syncthreads();
    double xi[RI], yi[RI], zi[RI], ax[RI], ay[RI], az[RI];
#pragma unroll
    for (int k = 0; k < RI; ++k) { xi[k] = 0.001 * (threadIdx.x + k * THREADS); yi[k] = 0.5 - xi[k]; zi[k] = 0.25 + 0.5 * xi[k]; ax[k] = ay[k] = az[k] = 0; }
    const long long t0 = clock64();
    for (int t = 0; t < ntiles; ++t) {
        if (ORDER == 0) {
#pragma unroll 1
            for (int j = 0; j < 256; j += 2) {
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const double2 XY = *reinterpret_cast<const double2*>(&T[j + q][0]), ZC = *reinterpret_cast<const double2*>(&T[j + q][2]);
#pragma unroll
                    for (int k = 0; k < RI; ++k) {
                        const double dX = fma(-xi[k], ZC.y, XY.x), dY = fma(-yi[k], ZC.y, XY.y), dZ = fma(-zi[k], ZC.y, ZC.x);
                        const double r2 = fma(dZ, dZ, fma(dY, dY, dX * dX));
                        const double y0 = seed64h(r2), y2 = y0 * y0, w = fma(r2, y2, -A), g = fma(w, w, C0), q3 = y0 * y2, s = q3 * g;
                        ax[k] = fma(dX, s, ax[k]); ay[k] = fma(dY, s, ay[k]); az[k] = fma(dZ, s, az[k]);
                    }
                }
            }
        } else {
            const double* src = &T[0][0];
#pragma unroll 1
            for (int j = 0; j < 256; ++j) {
                double2 XY, ZC;
                if (ORDER == 2) {
                    XY = *reinterpret_cast<const double2*>(src); ZC = *reinterpret_cast<const double2*>(src + 2);
                    src += 4;
                } else {
                    XY = *reinterpret_cast<const double2*>(&T[j][0]); ZC = *reinterpret_cast<const double2*>(&T[j][2]);
                }
                double dX[RI], dY[RI], dZ[RI], r2[RI], y0[RI], y2[RI], w[RI];
                FENCE(zero, 0);
#pragma unroll
                for (int k = 0; k < RI; ++k) dX[k] = fma(-xi[k], ZC.y, XY.x);
#pragma unroll
                for (int k = 0; k < RI; ++k) dY[k] = fma(-yi[k], ZC.y, XY.y);
#pragma unroll
                for (int k = 0; k < RI; ++k) dZ[k] = fma(-zi[k], ZC.y, ZC.x);
                FENCE(zero, 1);
#pragma unroll
                for (int k = 0; k < RI; ++k) r2[k] = fma(dZ[k], dZ[k], fma(dY[k], dY[k], dX[k] * dX[k]));
#pragma unroll
                for (int k = 0; k < RI; ++k) y0[k] = seed64h(r2[k]);
#pragma unroll
                for (int k = 0; k < RI; ++k) { y2[k] = y0[k] * y0[k]; w[k] = fma(r2[k], y2[k], -A); y2[k] = y0[k] * y2[k]; w[k] = fma(w[k], w[k], C0); w[k] = y2[k] * w[k]; }
                FENCE(zero, 2);
#pragma unroll
                for (int k = 0; k < RI; ++k) { ax[k] = fma(dX[k], w[k], ax[k]); ay[k] = fma(dY[k], w[k], ay[k]); az[k] = fma(dZ[k], w[k], az[k]); }
            }
        }
    }
    const long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int k = 0; k < RI; ++k) s += ax[k] + ay[k] + az[k];
    out[blockIdx.x * THREADS + threadIdx.x] = s;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}

// ---- host --------------------------------------------------------------------------------------------------------------------
static double* g_in; static double* g_out; static long long* g_clk;
static double slowest()
{
    CK(cudaDeviceSynchronize());
    std::vector<long long> h(SMS); CK(cudaMemcpy(h.data(), g_clk, SMS * 8, cudaMemcpyDeviceToHost));
    double mx = 0; for (long long v : h) mx = v > mx ? (double)v : mx;
    return mx;
}
template <int PAT> static void run_pattern(const char* name)
{
    const int iters = 5000;
    pattern_kernel<PAT><<<SMS, THREADS>>>(g_in, g_out, 10, g_clk);
    pattern_kernel<PAT><<<SMS, THREADS>>>(g_in, g_out, iters, g_clk);
    const double n = iters * 64.0 * (THREADS / 128);
    const double c = slowest() / n;
    printf("pattern  %-58s %.3f clk  %5.1f %% of nominal\n", name, c, 200.0 / c);
}
template <int MODE> static void run_lds(const char* name, double base)
{
    const int iters = 20000;
    lds_kernel<MODE><<<SMS, THREADS>>>(g_in, g_out, 10, g_clk);
    lds_kernel<MODE><<<SMS, THREADS>>>(g_in, g_out, iters, g_clk);
    const double n = iters * 56.0 * (THREADS / 128);
    const double c = slowest() / n;
    printf("loads    %-58s %.3f clk  %5.1f %% of nominal  (+%.1f clk per pass per warp)\n", name, c, 200.0 / c, (c - base) * 56);
}
template <int ORDER> static void run_far(const char* name)
{
    const int ntiles = 200;
    far_kernel<ORDER><<<SMS, THREADS>>>(g_in, g_out, 2, g_clk, 0);
    far_kernel<ORDER><<<SMS, THREADS>>>(g_in, g_out, ntiles, g_clk, 0);
    const double ipc = (double)ntiles * 256 * 4 * THREADS / slowest();        // interactions per clk per SM
    printf("far body %-58s %.3f interactions/clk/SM  pipe occupancy %5.1f %%  = %4.1f %% of FP64 peak at F = 20\n", name, ipc,
           100.0 * ipc * 14 / 64.0, 100.0 * ipc * 20 / 128.0);
}
int main()
{
    std::vector<double> h(2048);
    srand(7);
    for (int j = 0; j < 256; ++j) {            // a tile of sources away from the i-particles, (X, Y, Z, c) per source
        const double c = 1.0 + 0.5 * rand() / RAND_MAX;
        h[4 * j + 3] = c; h[4 * j] = c * (3.0 + 2.0 * rand() / RAND_MAX); h[4 * j + 1] = c * (-3.0 - 2.0 * rand() / RAND_MAX); h[4 * j + 2] = c * (4.0 * rand() / RAND_MAX);
    }
    for (int i = 1024; i < 2048; ++i) h[i] = 1.0 + 1e-9 * i;
    CK(cudaMalloc(&g_in, 2048 * 8)); CK(cudaMemcpy(g_in, h.data(), 2048 * 8, cudaMemcpyHostToDevice));
    CK(cudaMalloc(&g_out, SMS * THREADS * 8)); CK(cudaMalloc(&g_clk, SMS * 8));
    run_pattern<0>("DMUL  a_i = a_i * b0");
    run_pattern<1>("DFMA  a_i = b_i * b_i + a_i        (2 distinct registers)");
    run_pattern<2>("DFMA  a_i = b_i * c_i + a_i        (3 distinct, nothing to reuse)");
    run_pattern<3>("DFMA  a_i = b_i * c0 + a_i         (3 distinct, c0 reusable)");
    run_pattern<4>("DFMA  a_i = a_i * b0 + c0          (3 distinct, b0 and c0 reusable)");
    run_lds<0>("56 two-source DFMA per pass", 2.0);
    run_lds<1>("56 two-source DFMA + 4 LDS.64 per pass", 2.0);
    run_lds<2>("56 two-source DFMA + 2 LDS.128 per pass", 2.0);
    run_far<0>("14 instr, 2 sources x 4 i per pass, free order");
    run_far<1>("14 instr, 1 source x 4 i per pass, staged with fences");
    run_far<2>("14 instr, staged with fences, uniform-register LDS address");
    return 0;
}
