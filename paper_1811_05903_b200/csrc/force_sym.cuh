// force_sym.cuh -- the pair-symmetric force driver: every unordered FAR pair is evaluated ONCE and applied to both
// particles (Newton's third law; PAPER.md L131 counts the cost of the force calculation as N(N-1)/2 pair evaluations).
//
// Rows a1 + a3 of the hot path (Eq. 8 L88 first term, Eq. 4 third case L59) for the bulk of the pairs:
//
//   * The particles are cut into BLOCKS of IB = 2048 consecutive (radially sorted) particles = 8 j-tiles.  A block pair
//     (b, c) is "far" when the radial intervals of the two blocks are separated by more than hmax_b + hmax_c (the same
//     triangle-inequality test as tile_is_far, on block bounds): then no pair of it can be softened and every pair
//     is exactly Newtonian.  edge[b] = the last block that is not far from block b or from an earlier row (sym_band_width +
//     sym_plan_finalize, on the device; SymPlan in force_driver.cuh): for radially sorted input edge[b] - b = 1 ... 7
//     (N = 131,072 ... 1,048,576: the softening shell spans more of the ever thinner radial blocks) and differs from row to
//     row, for unsorted input edge[b] = nb - 1.
//   * Block pairs (b, c), b <= c <= edge[b], and their mirror images (the "band": the diagonal, all softened pairs, the self
//     pairs) go through the asymmetric persistent kernel of force_driver.cuh, restricted to the band's tiles.
//   * Every block pair with c > edge[b] is ONE work item of forces_sym_kernel: the CTA's 16 warps hold the 2048 particles of
//     block b in registers (4 per lane, as the asymmetric kernel does), block c's scaled sources sit in shared memory, and
//     warp w meets the sixteen 128-source subgroups of c in the order (w + q) mod 16, q = 0..15 (one __syncthreads per
//     round, so each subgroup's reaction sums in shared memory have one owner at a time).  Inside a (warp, subgroup)
//     meeting the sources are handed round the warp: at step s lane l works on source (l - s) mod 32 of the current
//     32-source set against its own 4 particles and then passes that source's reaction sums (3 doubles, 6 SHFL) on to
//     lane l + 1; after 32 steps every source has met all 128 particles of the warp and its sums are back in the
//     lane they started in.
//   * Per pair: 3 DFMA differences, 3 for r^2, 5 for r^-3 (the body of force_fp64.cuh), 1 DMUL s_i = m_i s and
//     2 x 3 DFMA accumulates = 18 FP64-pipe instructions per UNORDERED pair = 9 per ordered interaction (14 in the
//     asymmetric body).  The seven instructions of the accumulate stage are ordered so that each reads at most two new
//     register operands (w, then dZ, then s_i stay in the operand-reuse cache), i.e. all hold the pipe for 2 clk.
//   * An item writes two partial records of 3 x 2048 doubles: the forces of c on the particles of b (row record) and of b on
//     the particles of c (column record: the reaction sums B_j = sum_i m_i s dX times -1.875 c_j^2 = -1/m_j, see below).
//     forces_sym_reduce_kernel adds the records of each particle in fixed order (TwoSum, double-double) to the band's
//     result: bit-reproducible, no atomics.  Record memory is bounded by running the items in panels.
//
// Scaled sources (common.cuh): dX = X_j - c_j x_i = c_j (x_j - x_i), s = (c_j r)^-3 / 1.875, c_j = (1.875 m_j)^(-1/2):
//   force per unit mass on i:  m_j (x_j - x_i) / r^3 = s dX
//   force per unit mass on j:  m_i (x_i - x_j) / r^3 = -(m_i s dX) / m_j = -(1.875 c_j^2) (m_i s) dX
// Massless or unscalable particles cannot take part (their reaction sum cannot be divided by m_j): prep_tiles marks their
// tile hmax = +inf, which makes every block pair of that block "not far", W = nb - 1, and the whole evaluation runs
// through the asymmetric kernel -- slower, never wrong.
#pragma once
#include "common.cuh"
#include "force_fp64.cuh"
#include "force_mixed.cuh"
#include "force_driver.cuh"

namespace steps {

constexpr int TPB = IB / TJ;                 // j-tiles per block (8)
constexpr int SUBGROUPS = CTA_THREADS / 32;  // 128-particle subgroups per block = warps per CTA (16)
static_assert(IB % TJ == 0 && WARP_I * SUBGROUPS == IB, "block = whole tiles = one subgroup per warp");

// SymPlan (the device-resident plan of one force evaluation) is declared in force_driver.cuh.
__host__ __device__ inline long long sym_row_start(long long b, long long Km) { return b * Km - b * (b - 1) / 2; }

struct BlockMeta {
    float rmin, rmax, hmax;
};
template <typename Tile>
__device__ __forceinline__ BlockMeta block_meta(const Tile* __restrict__ tiles, int b)
{
    BlockMeta m{__int_as_float(0x7f800000), 0.0f, 0.0f};
#pragma unroll
    for (int t = 0; t < TPB; ++t) {
        const TileMeta tm = tiles[(long long)b * TPB + t].meta;
        m.rmin = fminf(m.rmin, tm.rmin); m.rmax = fmaxf(m.rmax, tm.rmax); m.hmax = fmaxf(m.hmax, tm.hmax);
    }
    return m;
}

// edge[b] (raw) = the last block c >= b that is not far from block b; plan->W = the largest c - b (plan->W must be 0 on
// entry: prep_tiles resets it).
template <typename Tile>
__global__ void __launch_bounds__(128) sym_band_width(const Tile* __restrict__ tiles, int nb, SymPlan* __restrict__ plan)
{
    const int b = blockIdx.x;
    const BlockMeta I = block_meta(tiles, b);
    int last = b;
    for (int c = b + 1 + threadIdx.x; c < nb; c += blockDim.x) {
        const BlockMeta J = block_meta(tiles, c);
        const TileMeta Jm{J.rmin, J.rmax, J.hmax, 0.0f};
        if (!tile_is_far(I.rmin, I.rmax, I.hmax, Jm)) last = max(last, c);
    }
    // a block that holds massless or unscalable particles (hmax = +inf) is not far from anything, ITSELF included: its own
    // row must reach the last block too
    if (!(I.hmax < __int_as_float(0x7f800000))) last = nb - 1;
    __shared__ int wmax[4];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = last;
    __syncthreads();
    if (threadIdx.x == 0) {
        last = max(max(wmax[0], wmax[1]), max(wmax[2], wmax[3]));
        const_cast<int*>(plan_edge(plan, nb))[b] = last;
        if (last > b) atomicMax(&plan->W, last - b);
    }
}

// One CTA: the plan's arrays.  per_row != 0: edge[] holds sym_band_width's raw edges (made non-decreasing here);
// per_row == 0: every row's band is plan->W blocks to either side (the periodic routes: W = 0, every block pair an item).
__global__ void __launch_bounds__(1024) sym_plan_finalize(SymPlan* __restrict__ plan, int nb, int sym_min_items, int split, int per_row)
{
    long long* cum = reinterpret_cast<long long*>(plan + 1);
    long long* rowstart = cum + nb + 1;
    int* edge = reinterpret_cast<int*>(rowstart + nb + 1);
    int* lo = edge + nb;
    __shared__ long long part[1024], part2[1024];
    __shared__ int pmax[1024];
    __shared__ int all_band;
    const int per = (nb + blockDim.x - 1) / blockDim.x;
    const int b0 = min(nb, (int)threadIdx.x * per), b1 = min(nb, b0 + per);
    const int W0 = plan->W;
    auto raw = [&](int b) { return per_row ? edge[b] : min(nb - 1, b + W0); };

    // running maximum of the raw edges: chunk maxima, their exclusive scan (thread 0), then each chunk again
    int m = 0;
    for (int b = b0; b < b1; ++b) m = max(m, raw(b));
    pmax[threadIdx.x] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int t = 0; t < (int)blockDim.x; ++t) { const int v = pmax[t]; pmax[t] = run; run = max(run, v); }
    }
    __syncthreads();
    m = pmax[threadIdx.x];
    long long items = 0;
    for (int b = b0; b < b1; ++b) { m = max(m, raw(b)); edge[b] = m; items += nb - 1 - m; }
    part[threadIdx.x] = items;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long K = 0;
        for (int t = 0; t < (int)blockDim.x; ++t) K += part[t];
        // too few items to balance over the SMs: everything through the band
        all_band = K * split < sym_min_items ? 1 : 0;
    }
    __syncthreads();
    if (all_band)
        for (int b = b0; b < b1; ++b) edge[b] = nb - 1;
    __syncthreads();                                          // edge[] complete (global writes of this CTA, read below)

    // lo[c] = the first row whose edge reaches c (edge[] is non-decreasing, edge[c] >= c)
    for (int c = b0; c < b1; ++c) {
        int l = 0, h = c;
        while (l < h) {
            const int mid = (l + h) >> 1;
            if (edge[mid] >= c) h = mid; else l = mid + 1;
        }
        lo[c] = l;
    }
    __syncthreads();
    long long s = 0;
    items = 0;
    int wmax = 0;
    for (int b = b0; b < b1; ++b) { s += (long long)(edge[b] - lo[b] + 1) * TPB; items += nb - 1 - edge[b]; wmax = max(wmax, edge[b] - b); }
    part[threadIdx.x] = s; part2[threadIdx.x] = items; pmax[threadIdx.x] = wmax;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long run = 0, run2 = 0;
        int W = 0;
        for (int t = 0; t < (int)blockDim.x; ++t) {
            const long long v = part[t], v2 = part2[t];
            part[t] = run; part2[t] = run2; run += v; run2 += v2; W = max(W, pmax[t]);
        }
        cum[nb] = run; rowstart[nb] = run2;
        plan->W = W; plan->nb = nb; plan->nt = nb * TPB; plan->K = run2; plan->T = run;
        plan->Km = nb > 0 ? lo[nb - 1] : 0;                  // rows before the first one whose band reaches the last block
    }
    __syncthreads();
    s = part[threadIdx.x]; items = part2[threadIdx.x];
    for (int b = b0; b < b1; ++b) {
        cum[b] = s; rowstart[b] = items;
        s += (long long)(edge[b] - lo[b] + 1) * TPB; items += nb - 1 - edge[b];
    }
}

__host__ __device__ constexpr int sym_smem_bytes() { return 2 * IB * (int)sizeof(FarSrcF64) + 3 * IB * (int)sizeof(double); }
#ifndef STEPS_SYM_FP64_THREADS
#define STEPS_SYM_FP64_THREADS 512
#endif
constexpr int SYM_FP64_THREADS = STEPS_SYM_FP64_THREADS;
constexpr int SYM_FP64_RI = IB / SYM_FP64_THREADS;

// Items [k_begin, k_end) of the plan's item list (one panel), shared out evenly over the grid.
// rowrec / colrec: [k - k_begin][3][IB] doubles.  THREADS x RI = 2,048: THREADS / 32 warps hold the block, RI particles per lane.
// SPLIT = false: one work unit per item (`split_arg` ignored, every loop bound a compile-time constant: the large-N kernel).
template <int THREADS, int RI, bool SPLIT>
__global__ void __launch_bounds__(THREADS, 1)
forces_sym_kernel(const TileF64* __restrict__ tiles, const SymPlan* __restrict__ plan, long long k_begin, long long k_end,
                  double* __restrict__ rowrec, double* __restrict__ colrec, int zero, int split_arg, int share_rank = 0,
                  int share_world = 1)
{
    const int split = SPLIT ? split_arg : 1;
    static_assert(THREADS * RI == IB, "the CTA holds one block");
    constexpr int WI = 32 * RI;                 // particles per warp = sources per subgroup
    constexpr int SUBG = THREADS / 32;          // warps = subgroups per block
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[2];
    FarSrcF64* col = reinterpret_cast<FarSrcF64*>(smem_raw);                       // [2][IB]
    double* Bsm = reinterpret_cast<double*>(smem_raw + 2 * IB * sizeof(FarSrcF64));   // [3][IB]

    // `split` parts per item (the SUBG rounds of an item shared among `split` consecutive sub-items, so that a mid-size N
    // still has enough work units for 148 SMs); [k_begin, k_end), the records and the grid's shares are in SUB-items
    // share_world > 1 (steps_forces_share): [k_begin, k_end) counts from the start of this rank's share of the sub-items
    const long long Kall = plan->K * split, S0 = Kall * share_rank / share_world, K = Kall * (share_rank + 1) / share_world;
    k_begin += S0; k_end += S0;
    if (k_end > K) k_end = K;
    if (k_begin >= k_end) return;
    const int nb = plan->nb;
    const long long n_items = k_end - k_begin;
    const long long kk0 = k_begin + (long long)blockIdx.x * n_items / gridDim.x;
    const long long kk1 = k_begin + ((long long)blockIdx.x + 1) * n_items / gridDim.x;
    const int total = (int)(kk1 - kk0);
    if (total <= 0) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // decode the first item: row b = the largest b with rowstart[b] <= kk0
    int b, c;
    {
        const int2 bc = sym_item_decode(plan, kk0 / split);
        b = bc.x; c = bc.y;
    }

    if (threadIdx.x == 0) {
        mbar_init(&full_bar[0], 1); mbar_init(&full_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // producer cursor (thread 0): the column block of item `it` goes to stage it & 1 by TPB bulk copies of the tiles' far[]
    int pb = b, pc = c;
    auto produce = [&](int it) {
        const int s = it & 1;
        mbar_expect_tx(&full_bar[s], (uint32_t)(IB * sizeof(FarSrcF64)));
#pragma unroll
        for (int t = 0; t < TPB; ++t)
            bulk_load(col + (size_t)s * IB + t * TJ, &tiles[(long long)pc * TPB + t].far[0], (uint32_t)(TJ * sizeof(FarSrcF64)),
                      &full_bar[s]);
        if ((kk0 + it + 1) % split == 0 && ++pc == nb) { ++pb; pc = sym_row_first_col(plan, pb); }     // the next sub-item starts a new item
    };
    if (threadIdx.x == 0) {
        produce(0);
        if (total > 1) produce(1);
    }

    constexpr double A = 1.4;
    constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);
    double xi[RI], yi[RI], zi[RI], mi[RI];
    int cur_b = -1;
    const int src_lane = (lane + 31) & 31;                       // reaction sums come from lane - 1

    for (int it = 0; it < total; ++it) {
        if (b != cur_b) {                                        // the row block's particles (plain copy of the tiles; pads: m = 0)
            cur_b = b;
#pragma unroll
            for (int k = 0; k < RI; ++k) {
                const int i = warp * WI + lane + 32 * k;     // within the block
                const TileF64& T = tiles[(long long)b * TPB + i / TJ];
                xi[k] = T.x[i % TJ]; yi[k] = T.y[i % TJ]; zi[k] = T.z[i % TJ]; mi[k] = T.m[i % TJ];
            }
        }
        double ax[RI], ay[RI], az[RI];
#pragma unroll
        for (int k = 0; k < RI; ++k) ax[k] = ay[k] = az[k] = 0.0;
        for (int q = threadIdx.x; q < 3 * IB; q += THREADS) Bsm[q] = 0.0;
        const int s = it & 1;
        mbar_wait(&full_bar[s], (it >> 1) & 1);
        __syncthreads();
        const FarSrcF64* cs = col + (size_t)s * IB;

        const int part = SPLIT ? (int)((kk0 + it) % split) : 0, rounds = SPLIT ? SUBG / split : SUBG;
        for (int q = part * rounds; q < (part + 1) * rounds; ++q) {
            const int u = (warp + q) & (SUBG - 1);
            for (int t = 0; t < WI / 32; ++t) {
                const FarSrcF64* set = cs + u * WI + t * 32;
                double bx = 0.0, by = 0.0, bz = 0.0;
                // (a 16-byte-half swizzle of the records removes the 2-way bank conflict of this 32-byte stride, but
                // its address arithmetic costs more than the conflict: measured 85.3 % against 87.1 % of peak)
#pragma unroll 1
                for (int st = 0; st < 32; ++st) {
                    // (loading the next step's source one step ahead costs 7 points: 79.7 % against 87.1 % of peak)
                    const FarSrcF64* src = set + ((lane - st) & 31);
                    const double2 XY = *reinterpret_cast<const double2*>(&src->X);
                    const double2 ZC = *reinterpret_cast<const double2*>(&src->Z);
                    const double X = XY.x, Y = XY.y, Z = ZC.x, C = ZC.y;
                    double dX[RI], dY[RI], dZ[RI], r2[RI], y0[RI], y2[RI], w[RI];
                    STEPS_STAGE_FENCE(zero, 0);
#pragma unroll
                    for (int k = 0; k < RI; ++k) dX[k] = fma(-xi[k], C, X);
#pragma unroll
                    for (int k = 0; k < RI; ++k) dY[k] = fma(-yi[k], C, Y);
#pragma unroll
                    for (int k = 0; k < RI; ++k) dZ[k] = fma(-zi[k], C, Z);
                    STEPS_STAGE_FENCE(zero, 1);
#pragma unroll
                    for (int k = 0; k < RI; ++k) r2[k] = fma(dZ[k], dZ[k], fma(dY[k], dY[k], dX[k] * dX[k]));
#pragma unroll
                    for (int k = 0; k < RI; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
                    for (int k = 0; k < RI; ++k) {
                        y2[k] = y0[k] * y0[k];
                        w[k] = fma(r2[k], y2[k], -A);
                        y2[k] = y0[k] * y2[k];
                        w[k] = fma(w[k], w[k], C0);
                        w[k] = y2[k] * w[k];
                    }
                    STEPS_STAGE_FENCE(zero, 2);
#pragma unroll
                    for (int k = 0; k < RI; ++k) {
                        // one basic block per particle: w, then dZ, then s_i stay in the operand-reuse cache, every instruction
                        // reads at most two new operands (ptxas otherwise hoists the s_i products: 85.1 -> 87.1 % of peak)
                        if (k > 0) STEPS_STAGE_FENCE(zero, 2 + k);
                        const double si = mi[k] * w[k];
                        ax[k] = fma(dX[k], w[k], ax[k]);
                        ay[k] = fma(dY[k], w[k], ay[k]);
                        az[k] = fma(dZ[k], w[k], az[k]);
                        bz = fma(dZ[k], si, bz);
                        by = fma(dY[k], si, by);
                        bx = fma(dX[k], si, bx);
                    }
                    bx = __shfl_sync(0xffffffffu, bx, src_lane);
                    by = __shfl_sync(0xffffffffu, by, src_lane);
                    bz = __shfl_sync(0xffffffffu, bz, src_lane);
                }
                // 32 hand-overs later the sums of source `lane` of the set are back in this lane
                const int j = u * WI + t * 32 + lane;
                Bsm[j] += bx; Bsm[IB + j] += by; Bsm[2 * IB + j] += bz;
            }
            __syncthreads();
        }

        // partial records of the item
        const long long rec = (kk0 + it - k_begin) * 3 * IB;
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            const int i = warp * WI + lane + 32 * k;
            rowrec[rec + i] = ax[k]; rowrec[rec + IB + i] = ay[k]; rowrec[rec + 2 * IB + i] = az[k];
        }
        for (int j = threadIdx.x; j < IB; j += THREADS) {
            const double cj = cs[j].c;
            const double f = -STEPS_FP64_FOLD * cj * cj;
            colrec[rec + j] = f * Bsm[j]; colrec[rec + IB + j] = f * Bsm[IB + j]; colrec[rec + 2 * IB + j] = f * Bsm[2 * IB + j];
        }
        __syncthreads();                                          // stage s and Bsm are free again
        if (threadIdx.x == 0 && it + 2 < total) produce(it + 2);
        if ((kk0 + it + 1) % split == 0 && ++c == nb) { ++b; c = sym_row_first_col(plan, b); }
    }
}

// ---- the same for the MIXED path (fp32 pairs, fp64 accumulation) ------------------------------------------------------
// Per step a lane meets one source with its 4 particles packed in two pairs (FFMA2 / FMUL2, the source's scalars broadcast to
// both halves): per packed pair 3 differences, 3 for r^2, 2 MUFU.RSQ, 2 for y^3, 1 for s_i = m_i y^3 and 2 x 3 accumulates
// = 15 packed FP32-pipe instructions + 2 MUFU per FOUR ordered interactions (11 + 2 per two in the asymmetric body).
// fp32 sums never hold more than 128 terms: the particles' sums are flushed into fp64 accumulators in shared memory after
// every 128-source subgroup, the sources' reaction sums (two packed halves, 64 terms each) into fp64 shared memory after the
// 32 hand-overs of a set.  Scaled sources: c_j = m_j^(-1/2) in fp32, dX = X_j - c_j x_i, y = 1/(c_j r):
//   on i:  m_j (x_j - x_i)/r^3 = y^3 dX          on j:  -(m_i y^3 dX) c_j^2
// THREADS x RI = 2,048: the block is held by THREADS / 32 warps with RI particles per lane.  More particles per lane means
// more packed arithmetic per hand-over (the shuffles and the source load are per step, whatever RI is).
__host__ __device__ constexpr int sym_mixed_stage_bytes() { return TPB * 4 * TJ * (int)sizeof(float); }     // (X, Y, Z, c) of the block's tiles
template <int THREADS, int RI>
__host__ __device__ constexpr int sym_mixed_smem_bytes()
{
    return 2 * sym_mixed_stage_bytes() + 3 * IB * (int)sizeof(double) + 3 * RI * THREADS * (int)sizeof(double);
}
#ifndef STEPS_SYM_MIXED_THREADS
#define STEPS_SYM_MIXED_THREADS 256
#endif
constexpr int SYM_MIXED_THREADS = STEPS_SYM_MIXED_THREADS;
constexpr int SYM_MIXED_RI = IB / SYM_MIXED_THREADS;

template <int THREADS, int RI, bool SPLIT>
__global__ void __launch_bounds__(THREADS, 1)
forces_sym_mixed_kernel(const TileF32* __restrict__ tiles, const SymPlan* __restrict__ plan, long long k_begin, long long k_end,
                        double* __restrict__ rowrec, double* __restrict__ colrec, int split_arg, int share_rank = 0, int share_world = 1)
{
    const int split = SPLIT ? split_arg : 1;
    static_assert(THREADS * RI == IB && RI % 2 == 0, "the CTA holds one block, particles packed in pairs");
    constexpr int NP = RI / 2;                  // packed pairs per lane
    constexpr int WI = 32 * RI;                 // particles per warp = sources per subgroup
    constexpr int SUBG = THREADS / 32;          // warps = subgroups per block
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[2];
    constexpr int STAGE = sym_mixed_stage_bytes();
    float* col = reinterpret_cast<float*>(smem_raw);                                   // [2][TPB][4][TJ]
    double* Bsm = reinterpret_cast<double*>(smem_raw + 2 * STAGE);                     // [3][IB]
    double* Asm = Bsm + 3 * IB + threadIdx.x;                                          // [3][RI][THREADS], this thread's column

    // `split` parts per item (the SUBG rounds of an item shared among `split` consecutive sub-items, so that a mid-size N
    // still has enough work units for 148 SMs); [k_begin, k_end), the records and the grid's shares are in SUB-items
    // share_world > 1 (steps_forces_share): [k_begin, k_end) counts from the start of this rank's share of the sub-items
    const long long Kall = plan->K * split, S0 = Kall * share_rank / share_world, K = Kall * (share_rank + 1) / share_world;
    k_begin += S0; k_end += S0;
    if (k_end > K) k_end = K;
    if (k_begin >= k_end) return;
    const int nb = plan->nb;
    const long long n_items = k_end - k_begin;
    const long long kk0 = k_begin + (long long)blockIdx.x * n_items / gridDim.x;
    const long long kk1 = k_begin + ((long long)blockIdx.x + 1) * n_items / gridDim.x;
    const int total = (int)(kk1 - kk0);
    if (total <= 0) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int b, c;
    {
        const int2 bc = sym_item_decode(plan, kk0 / split);
        b = bc.x; c = bc.y;
    }
    if (threadIdx.x == 0) {
        mbar_init(&full_bar[0], 1); mbar_init(&full_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int pb = b, pc = c;
    auto produce = [&](int it) {
        const int s = it & 1;
        mbar_expect_tx(&full_bar[s], (uint32_t)STAGE);
#pragma unroll
        for (int t = 0; t < TPB; ++t)          // X[], Y[], Z[], c[] are the first 4 TJ floats of a tile record
            bulk_load(reinterpret_cast<unsigned char*>(col) + (size_t)s * STAGE + t * (4 * TJ * sizeof(float)),
                      &tiles[(long long)pc * TPB + t].X[0], (uint32_t)(4 * TJ * sizeof(float)), &full_bar[s]);
        if ((kk0 + it + 1) % split == 0 && ++pc == nb) { ++pb; pc = sym_row_first_col(plan, pb); }     // the next sub-item starts a new item
    };
    if (threadIdx.x == 0) {
        produce(0);
        if (total > 1) produce(1);
    }

    u64 nx[NP], ny[NP], nz[NP], m2[NP];
    int cur_b = -1;
    const int src_lane = (lane + 31) & 31;

    for (int it = 0; it < total; ++it) {
        if (b != cur_b) {
            cur_b = b;
            float x[RI], y[RI], z[RI], m[RI];
#pragma unroll
            for (int k = 0; k < RI; ++k) {
                const int i = warp * WI + lane + 32 * k;
                const TileF32& T = tiles[(long long)b * TPB + i / TJ];
                x[k] = T.x[i % TJ]; y[k] = T.y[i % TJ]; z[k] = T.z[i % TJ]; m[k] = T.m[i % TJ];
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                nx[p] = pack2(-x[2 * p], -x[2 * p + 1]); ny[p] = pack2(-y[2 * p], -y[2 * p + 1]);
                nz[p] = pack2(-z[2 * p], -z[2 * p + 1]); m2[p] = pack2(m[2 * p], m[2 * p + 1]);
            }
        }
#pragma unroll
        for (int q = 0; q < 3 * RI; ++q) Asm[q * THREADS] = 0.0;
        for (int q = threadIdx.x; q < 3 * IB; q += THREADS) Bsm[q] = 0.0;
        const int s = it & 1;
        mbar_wait(&full_bar[s], (it >> 1) & 1);
        __syncthreads();
        const float* cs = col + (size_t)s * (STAGE / sizeof(float));

        const int part = SPLIT ? (int)((kk0 + it) % split) : 0, rounds = SPLIT ? SUBG / split : SUBG;
        for (int q = part * rounds; q < (part + 1) * rounds; ++q) {
            const int u = (warp + q) & (SUBG - 1);
            u64 ax[NP], ay[NP], az[NP];
#pragma unroll
            for (int p = 0; p < NP; ++p) ax[p] = ay[p] = az[p] = 0ull;
            for (int t = 0; t < WI / 32; ++t) {
                const int j0 = u * WI + t * 32;                                       // first source of the set (within the block)
                const float* set = cs + (j0 / TJ) * (4 * TJ) + (j0 % TJ);           // X of source j0; Y, Z, c follow at + TJ each
                u64 bx = 0ull, by = 0ull, bz = 0ull;
#pragma unroll 2
                for (int st = 0; st < 32; ++st) {
                    const int r = (lane - st) & 31;
                    const float X = set[r], Y = set[TJ + r], Z = set[2 * TJ + r], C = set[3 * TJ + (r ^ STEPS_C_SWIZZLE)];
                    const u64 cq = pack2(C, C), Xq = pack2(X, X), Yq = pack2(Y, Y), Zq = pack2(Z, Z);
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        const u64 dX = fma2(nx[p], cq, Xq), dY = fma2(ny[p], cq, Yq), dZ = fma2(nz[p], cq, Zq);
                        const u64 r2 = fma2(dZ, dZ, fma2(dY, dY, mul2(dX, dX)));
                        float ra, rb;
                        unpack2(r2, ra, rb);
                        const u64 y = pack2(rsqrt_approx(ra), rsqrt_approx(rb));
                        const u64 y3 = mul2(mul2(y, y), y);
                        const u64 si = mul2(y3, m2[p]);
                        ax[p] = fma2(dX, y3, ax[p]);
                        ay[p] = fma2(dY, y3, ay[p]);
                        az[p] = fma2(dZ, y3, az[p]);
                        bz = fma2(dZ, si, bz);
                        by = fma2(dY, si, by);
                        bx = fma2(dX, si, bx);
                    }
                    bx = __shfl_sync(0xffffffffu, bx, src_lane);
                    by = __shfl_sync(0xffffffffu, by, src_lane);
                    bz = __shfl_sync(0xffffffffu, bz, src_lane);
                }
                float lo, hi;
                const int j = j0 + lane;                       // 32 steps x NP terms per packed half: <= 128
                unpack2(bx, lo, hi); Bsm[j] += (double)lo + (double)hi;
                unpack2(by, lo, hi); Bsm[IB + j] += (double)lo + (double)hi;
                unpack2(bz, lo, hi); Bsm[2 * IB + j] += (double)lo + (double)hi;
                if ((t & 3) == 3) {                            // 128 sources per particle: into the fp64 accumulators
#pragma unroll
                    for (int p = 0; p < NP; ++p) {
                        unpack2(ax[p], lo, hi); Asm[(0 * RI + 2 * p) * THREADS] += (double)lo; Asm[(0 * RI + 2 * p + 1) * THREADS] += (double)hi;
                        unpack2(ay[p], lo, hi); Asm[(1 * RI + 2 * p) * THREADS] += (double)lo; Asm[(1 * RI + 2 * p + 1) * THREADS] += (double)hi;
                        unpack2(az[p], lo, hi); Asm[(2 * RI + 2 * p) * THREADS] += (double)lo; Asm[(2 * RI + 2 * p + 1) * THREADS] += (double)hi;
                        ax[p] = ay[p] = az[p] = 0ull;
                    }
                }
            }
            __syncthreads();
        }

        const long long rec = (kk0 + it - k_begin) * 3 * IB;
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            const int i = warp * WI + lane + 32 * k;
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) rowrec[rec + cc * IB + i] = Asm[(cc * RI + k) * THREADS];
        }
        for (int j = threadIdx.x; j < IB; j += THREADS) {
            const double cj = (double)cs[(j / TJ) * (4 * TJ) + 3 * TJ + ((j % TJ) ^ STEPS_C_SWIZZLE)];
            const double f = -cj * cj;
            colrec[rec + j] = f * Bsm[j]; colrec[rec + IB + j] = f * Bsm[IB + j]; colrec[rec + 2 * IB + j] = f * Bsm[2 * IB + j];
        }
        __syncthreads();
        if (threadIdx.x == 0 && it + 2 < total) produce(it + 2);
        if ((kk0 + it + 1) % split == 0 && ++c == nb) { ++b; c = sym_row_first_col(plan, b); }
    }
}

// ---- the pair-symmetric evaluation in a periodic box (leading image, Eq. 5) -------------
// The same items, rounds, hand-over and records as above, with three differences:
//   * every block pair (b, c), c > b, is an item (W = 0): in a periodic box closeness is not a matter of |c - b|.  Which
//     pairs may be softened is decided per MEETING of a warp's group (128 particles fp64 / 256 mixed) with a subgroup of
//     the column block, by pair_decision (common.cuh) on the groups' bounding boxes: a meeting that may hold a softened pair
//     is skipped here and evaluated by forces_boxring_kernel in restricted mode (force_driver.cuh), which takes the very
//     same decision from the very same call;
//   * the image shift of the meeting goes onto the warp's particles (a copy of the row block's positions stays in shared
//     memory, each thread's own four/eight), and the components whose separations straddle half the box are folded
//     (fold_f64 / fold2: one addition + one bit operation per pair and component), the body chosen by the fold mask;
//   * the reaction on j uses the folded separation as well -- the leading image of x_i - x_j is minus that of x_j - x_i.
// Hand-over of a column subgroup between the warps of the periodic symmetric kernels.  Warp w meets subgroup (w + q) mod SUBG
// in round q, so the subgroup it needs next was last used -- one round earlier -- by warp w + 1, and by nobody else: instead
// of a CTA-wide barrier per round (every round then costs what its most-folded meeting costs) a warp only waits for its
// neighbour's count of finished rounds.  The warps drift apart by a few rounds and the meetings' costs average out.
__device__ __forceinline__ void round_publish(int* counter, int value)      // one lane, after __syncwarp
{
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(smem_u32(counter)), "r"(value) : "memory");
}
__device__ __forceinline__ void round_wait(const int* counter, int value)   // one lane, followed by __syncwarp
{
    int seen;
    for (;;) {
        asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(seen) : "r"(smem_u32(counter)) : "memory");
        if (seen >= value) break;
        __nanosleep(200);                                    // a spinning warp would take issue slots from the working ones
    }
}

template <int RI, int MASK>
__device__ __forceinline__ void sym_box_steps(const FarSrcF64* __restrict__ set, int lane, int src_lane, const double (&xi)[RI],
                                              const double (&yi)[RI], const double (&zi)[RI], const double (&mi)[RI], double (&ax)[RI],
                                              double (&ay)[RI], double (&az)[RI], double& bx, double& by, double& bz, int zero, double halfL)
{
    constexpr double A = 1.4;
    constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);
#pragma unroll 1
    for (int st = 0; st < 32; ++st) {
        const FarSrcF64* src = set + ((lane - st) & 31);
        const double2 XY = *reinterpret_cast<const double2*>(&src->X);
        const double2 ZC = *reinterpret_cast<const double2*>(&src->Z);
        const double X = XY.x, Y = XY.y, Z = ZC.x, C = ZC.y;
        const double hc = C * halfL;
        double dX[RI], dY[RI], dZ[RI], r2[RI], y0[RI], y2[RI], w[RI];
        STEPS_STAGE_FENCE(zero, 0);
#pragma unroll
        for (int k = 0; k < RI; ++k) dX[k] = fma(-xi[k], C, X);
#pragma unroll
        for (int k = 0; k < RI; ++k) dY[k] = fma(-yi[k], C, Y);
#pragma unroll
        for (int k = 0; k < RI; ++k) dZ[k] = fma(-zi[k], C, Z);
        if (MASK & 1) {
#pragma unroll
            for (int k = 0; k < RI; ++k) dX[k] = fold_f64(dX[k], hc);
        }
        if (MASK & 2) {
#pragma unroll
            for (int k = 0; k < RI; ++k) dY[k] = fold_f64(dY[k], hc);
        }
        if (MASK & 4) {
#pragma unroll
            for (int k = 0; k < RI; ++k) dZ[k] = fold_f64(dZ[k], hc);
        }
        STEPS_STAGE_FENCE(zero, 1);
#pragma unroll
        for (int k = 0; k < RI; ++k) r2[k] = fma(dZ[k], dZ[k], fma(dY[k], dY[k], dX[k] * dX[k]));
#pragma unroll
        for (int k = 0; k < RI; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            y2[k] = y0[k] * y0[k];
            w[k] = fma(r2[k], y2[k], -A);
            y2[k] = y0[k] * y2[k];
            w[k] = fma(w[k], w[k], C0);
            w[k] = y2[k] * w[k];
        }
        STEPS_STAGE_FENCE(zero, 2);
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            if (k > 0) STEPS_STAGE_FENCE(zero, 2 + k);
            const double si = mi[k] * w[k];
            ax[k] = fma(dX[k], w[k], ax[k]);
            ay[k] = fma(dY[k], w[k], ay[k]);
            az[k] = fma(dZ[k], w[k], az[k]);
            bz = fma(dZ[k], si, bz);
            by = fma(dY[k], si, by);
            bx = fma(dX[k], si, bx);
        }
        bx = __shfl_sync(0xffffffffu, bx, src_lane);
        by = __shfl_sync(0xffffffffu, by, src_lane);
        bz = __shfl_sync(0xffffffffu, bz, src_lane);
    }
}

__host__ __device__ constexpr int sym_box_smem_bytes() { return sym_smem_bytes() + 3 * IB * (int)sizeof(double); }

template <int THREADS, int RI, bool SPLIT>
__global__ void __launch_bounds__(THREADS, 1)
forces_sym_box_kernel(const TileF64* __restrict__ tiles, const SymPlan* __restrict__ plan, const GroupMeta* __restrict__ gm,
                      long long k_begin, long long k_end, double* __restrict__ rowrec, double* __restrict__ colrec, int zero,
                      int split_arg, double box_L, double box_invL)
{
    const int split = SPLIT ? split_arg : 1;
    static_assert(THREADS * RI == IB, "the CTA holds one block");
    constexpr int WI = 32 * RI;                 // particles per warp = sources per subgroup
    constexpr int SUBG = THREADS / 32;          // warps = subgroups per block
    static_assert(WI == WARP_I, "a warp's particles are one group of GroupMeta");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[2];
    FarSrcF64* col = reinterpret_cast<FarSrcF64*>(smem_raw);                       // [2][IB]
    double* Bsm = reinterpret_cast<double*>(smem_raw + 2 * IB * sizeof(FarSrcF64));   // [3][IB]
    double* Xsm = Bsm + 3 * IB + threadIdx.x;                                      // [3][RI][THREADS]: the row block, unshifted
    __shared__ int round_done[SUBG];                                               // rounds finished per warp (round_wait)
    if (threadIdx.x < SUBG) round_done[threadIdx.x] = 0;

    const long long K = plan->K * split;
    if (k_end > K) k_end = K;
    if (k_begin >= k_end) return;
    const int nb = plan->nb, Km = plan->Km;     // W = 0: item (b, c) for every c > b
    const long long n_items = k_end - k_begin;
    const long long kk0 = k_begin + (long long)blockIdx.x * n_items / gridDim.x;
    const long long kk1 = k_begin + ((long long)blockIdx.x + 1) * n_items / gridDim.x;
    const int total = (int)(kk1 - kk0);
    if (total <= 0) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int b, c;
    {
        const double t = 2.0 * Km + 1.0;
        const long long item0 = kk0 / split;
        int bb = (int)((t - sqrt(fmax(t * t - 8.0 * (double)item0, 0.0))) * 0.5);
        bb = max(0, min(bb, Km - 1));
        while (bb + 1 < Km && sym_row_start(bb + 1, Km) <= item0) ++bb;
        while (bb > 0 && sym_row_start(bb, Km) > item0) --bb;
        b = bb;
        c = bb + 1 + (int)(item0 - sym_row_start(bb, Km));
    }

    if (threadIdx.x == 0) {
        mbar_init(&full_bar[0], 1); mbar_init(&full_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    int pb = b, pc = c;
    auto produce = [&](int it) {
        const int s = it & 1;
        mbar_expect_tx(&full_bar[s], (uint32_t)(IB * sizeof(FarSrcF64)));
#pragma unroll
        for (int t = 0; t < TPB; ++t)
            bulk_load(col + (size_t)s * IB + t * TJ, &tiles[(long long)pc * TPB + t].far[0], (uint32_t)(TJ * sizeof(FarSrcF64)),
                      &full_bar[s]);
        if ((kk0 + it + 1) % split == 0 && ++pc == nb) { ++pb; pc = pb + 1; }
    };
    if (threadIdx.x == 0) {
        produce(0);
        if (total > 1) produce(1);
    }

    double mi[RI];
    int cur_b = -1;
    const int src_lane = (lane + 31) & 31;
    const double halfL = 0.5 * box_L;

    for (int it = 0; it < total; ++it) {
        if (b != cur_b) {
            cur_b = b;
#pragma unroll
            for (int k = 0; k < RI; ++k) {
                const int i = warp * WI + lane + 32 * k;
                const TileF64& T = tiles[(long long)b * TPB + i / TJ];
                Xsm[(0 * RI + k) * THREADS] = T.x[i % TJ]; Xsm[(1 * RI + k) * THREADS] = T.y[i % TJ];
                Xsm[(2 * RI + k) * THREADS] = T.z[i % TJ]; mi[k] = T.m[i % TJ];
            }
        }
        double ax[RI], ay[RI], az[RI];
#pragma unroll
        for (int k = 0; k < RI; ++k) ax[k] = ay[k] = az[k] = 0.0;
        for (int q = threadIdx.x; q < 3 * IB; q += THREADS) Bsm[q] = 0.0;
        const int s = it & 1;
        mbar_wait(&full_bar[s], (it >> 1) & 1);
        __syncthreads();
        const FarSrcF64* cs = col + (size_t)s * IB;

        // the image decisions of this warp's SUBG meetings of the item, one per lane (boxcode_pack, force_driver.cuh)
        const uint32_t my_code = boxcode_pack(pair_decision<1>(gm, b * SUBG + warp, c * SUBG + (lane & (SUBG - 1)), box_L, box_invL), box_invL);
        const int part = SPLIT ? (int)((kk0 + it) % split) : 0, rounds = SPLIT ? SUBG / split : SUBG;
        const int base = it * rounds;                         // rounds every warp had finished when this item started
        for (int q = part * rounds; q < (part + 1) * rounds; ++q) {
            const int u = (warp + q) & (SUBG - 1);
            if (q > part * rounds) {                          // subgroup u was warp + 1's in the round before (round_wait above)
                if (lane == 0) round_wait(&round_done[(warp + 1) & (SUBG - 1)], base + (q - part * rounds));
                __syncwarp();
            }
            const BoxShift dec = boxcode_unpack(__shfl_sync(0xffffffffu, my_code, u), box_L);
            if (dec.kind != 0) {                              // else: forces_boxring_kernel evaluates this meeting
                double xi[RI], yi[RI], zi[RI];
#pragma unroll
                for (int k = 0; k < RI; ++k) {
                    xi[k] = Xsm[(0 * RI + k) * THREADS] + dec.s[0]; yi[k] = Xsm[(1 * RI + k) * THREADS] + dec.s[1];
                    zi[k] = Xsm[(2 * RI + k) * THREADS] + dec.s[2];
                }
                for (int t = 0; t < WI / 32; ++t) {
                    const FarSrcF64* set = cs + u * WI + t * 32;
                    double bx = 0.0, by = 0.0, bz = 0.0;
                    switch (dec.mask) {
                        case 0: sym_box_steps<RI, 0>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        case 1: sym_box_steps<RI, 1>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        case 2: sym_box_steps<RI, 2>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        case 3: sym_box_steps<RI, 3>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        case 4: sym_box_steps<RI, 4>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        case 5: sym_box_steps<RI, 5>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        case 6: sym_box_steps<RI, 6>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                        default: sym_box_steps<RI, 7>(set, lane, src_lane, xi, yi, zi, mi, ax, ay, az, bx, by, bz, zero, halfL); break;
                    }
                    const int j = u * WI + t * 32 + lane;
                    Bsm[j] += bx; Bsm[IB + j] += by; Bsm[2 * IB + j] += bz;
                }
            }
            __syncwarp();
            if (lane == 0) round_publish(&round_done[warp], base + (q - part * rounds) + 1);
        }
        __syncthreads();                                      // every subgroup's reaction sums are complete

        const long long rec = (kk0 + it - k_begin) * 3 * IB;
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            const int i = warp * WI + lane + 32 * k;
            rowrec[rec + i] = ax[k]; rowrec[rec + IB + i] = ay[k]; rowrec[rec + 2 * IB + i] = az[k];
        }
        for (int j = threadIdx.x; j < IB; j += THREADS) {
            const double cj = cs[j].c;
            const double f = -STEPS_FP64_FOLD * cj * cj;
            colrec[rec + j] = f * Bsm[j]; colrec[rec + IB + j] = f * Bsm[IB + j]; colrec[rec + 2 * IB + j] = f * Bsm[2 * IB + j];
        }
        __syncthreads();
        if (threadIdx.x == 0 && it + 2 < total) produce(it + 2);
        if ((kk0 + it + 1) % split == 0 && ++c == nb) { ++b; c = b + 1; }
    }
}

// The mixed path of the same: the warp's 256 particles are two groups of GroupMeta (pair_decision<2>), a subgroup is one tile.
template <int THREADS, int RI>
__host__ __device__ constexpr int sym_mixed_box_smem_bytes() { return sym_mixed_smem_bytes<THREADS, RI>() + 3 * IB * (int)sizeof(float); }

#ifndef STEPS_SYMBOX_UNROLL
#define STEPS_SYMBOX_UNROLL 1
#endif
template <int NP, int MASK>
__device__ __forceinline__ void sym_mixed_box_steps(const float* __restrict__ set, int lane, int src_lane, const u64 (&nx)[NP],
                                                    const u64 (&ny)[NP], const u64 (&nz)[NP], const u64 (&m2)[NP], u64 (&ax)[NP],
                                                    u64 (&ay)[NP], u64 (&az)[NP], u64& bx, u64& by, u64& bz, float halfL)
{
STEPS_UNROLL(STEPS_SYMBOX_UNROLL)
    for (int st = 0; st < 32; ++st) {
        const int r = (lane - st) & 31;
        const float X = set[r], Y = set[TJ + r], Z = set[2 * TJ + r], C = set[3 * TJ + (r ^ STEPS_C_SWIZZLE)];
        const u64 cq = pack2(C, C), Xq = pack2(X, X), Yq = pack2(Y, Y), Zq = pack2(Z, Z);
        const float hc = C * halfL;
        const u64 h2 = pack2(hc, hc);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            u64 dX = fma2(nx[p], cq, Xq), dY = fma2(ny[p], cq, Yq), dZ = fma2(nz[p], cq, Zq);
            if (MASK & 1) dX = MixedPath::fold2(dX, h2);
            if (MASK & 2) dY = MixedPath::fold2(dY, h2);
            if (MASK & 4) dZ = MixedPath::fold2(dZ, h2);
            const u64 r2 = fma2(dZ, dZ, fma2(dY, dY, mul2(dX, dX)));
            float ra, rb;
            unpack2(r2, ra, rb);
            const u64 y = pack2(rsqrt_approx(ra), rsqrt_approx(rb));
            const u64 y3 = mul2(mul2(y, y), y);
            const u64 si = mul2(y3, m2[p]);
            ax[p] = fma2(dX, y3, ax[p]);
            ay[p] = fma2(dY, y3, ay[p]);
            az[p] = fma2(dZ, y3, az[p]);
            bz = fma2(dZ, si, bz);
            by = fma2(dY, si, by);
            bx = fma2(dX, si, bx);
        }
        bx = __shfl_sync(0xffffffffu, bx, src_lane);
        by = __shfl_sync(0xffffffffu, by, src_lane);
        bz = __shfl_sync(0xffffffffu, bz, src_lane);
    }
}

template <int THREADS, int RI, bool SPLIT>
__global__ void __launch_bounds__(THREADS, 1)
forces_sym_mixed_box_kernel(const TileF32* __restrict__ tiles, const SymPlan* __restrict__ plan, const GroupMeta* __restrict__ gm,
                            long long k_begin, long long k_end, double* __restrict__ rowrec, double* __restrict__ colrec,
                            int split_arg, double box_L, double box_invL)
{
    const int split = SPLIT ? split_arg : 1;
    static_assert(THREADS * RI == IB && RI % 2 == 0, "the CTA holds one block, particles packed in pairs");
    constexpr int NP = RI / 2;                  // packed pairs per lane
    constexpr int WI = 32 * RI;                 // particles per warp = sources per subgroup
    constexpr int SUBG = THREADS / 32;          // warps = subgroups per block
    static_assert(WI == 2 * WARP_I && WI == TJ, "a warp's particles are two groups of GroupMeta, a subgroup is one tile");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[2];
    constexpr int STAGE = sym_mixed_stage_bytes();
    float* col = reinterpret_cast<float*>(smem_raw);                                   // [2][TPB][4][TJ]
    double* Bsm = reinterpret_cast<double*>(smem_raw + 2 * STAGE);                     // [3][IB]
    double* Asm = Bsm + 3 * IB + threadIdx.x;                                          // [3][RI][THREADS], this thread's column
    float* Xsm = reinterpret_cast<float*>(Bsm + 3 * IB + 3 * RI * THREADS) + threadIdx.x;   // [3][RI][THREADS]: the row block, unshifted

    const long long K = plan->K * split;
    if (k_end > K) k_end = K;
    if (k_begin >= k_end) return;
    const int nb = plan->nb, Km = plan->Km;
    const long long n_items = k_end - k_begin;
    const long long kk0 = k_begin + (long long)blockIdx.x * n_items / gridDim.x;
    const long long kk1 = k_begin + ((long long)blockIdx.x + 1) * n_items / gridDim.x;
    const int total = (int)(kk1 - kk0);
    if (total <= 0) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int b, c;
    {
        const double t = 2.0 * Km + 1.0;
        const long long item0 = kk0 / split;
        int bb = (int)((t - sqrt(fmax(t * t - 8.0 * (double)item0, 0.0))) * 0.5);
        bb = max(0, min(bb, Km - 1));
        while (bb + 1 < Km && sym_row_start(bb + 1, Km) <= item0) ++bb;
        while (bb > 0 && sym_row_start(bb, Km) > item0) --bb;
        b = bb;
        c = bb + 1 + (int)(item0 - sym_row_start(bb, Km));
    }
    if (threadIdx.x == 0) {
        mbar_init(&full_bar[0], 1); mbar_init(&full_bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int pb = b, pc = c;
    auto produce = [&](int it) {
        const int s = it & 1;
        mbar_expect_tx(&full_bar[s], (uint32_t)STAGE);
#pragma unroll
        for (int t = 0; t < TPB; ++t)
            bulk_load(reinterpret_cast<unsigned char*>(col) + (size_t)s * STAGE + t * (4 * TJ * sizeof(float)),
                      &tiles[(long long)pc * TPB + t].X[0], (uint32_t)(4 * TJ * sizeof(float)), &full_bar[s]);
        if ((kk0 + it + 1) % split == 0 && ++pc == nb) { ++pb; pc = pb + 1; }
    };
    if (threadIdx.x == 0) {
        produce(0);
        if (total > 1) produce(1);
    }

    u64 m2[NP];
    int cur_b = -1;
    const int src_lane = (lane + 31) & 31;
    const float halfL = (float)(0.5 * box_L);

    for (int it = 0; it < total; ++it) {
        if (b != cur_b) {
            cur_b = b;
            float m[RI];
#pragma unroll
            for (int k = 0; k < RI; ++k) {
                const int i = warp * WI + lane + 32 * k;
                const TileF32& T = tiles[(long long)b * TPB + i / TJ];
                Xsm[(0 * RI + k) * THREADS] = T.x[i % TJ]; Xsm[(1 * RI + k) * THREADS] = T.y[i % TJ];
                Xsm[(2 * RI + k) * THREADS] = T.z[i % TJ]; m[k] = T.m[i % TJ];
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) m2[p] = pack2(m[2 * p], m[2 * p + 1]);
        }
#pragma unroll
        for (int q = 0; q < 3 * RI; ++q) Asm[q * THREADS] = 0.0;
        for (int q = threadIdx.x; q < 3 * IB; q += THREADS) Bsm[q] = 0.0;
        const int s = it & 1;
        mbar_wait(&full_bar[s], (it >> 1) & 1);
        __syncthreads();
        const float* cs = col + (size_t)s * (STAGE / sizeof(float));

        const uint32_t my_code = boxcode_pack(pair_decision<2>(gm, b * SUBG + warp, c * SUBG + (lane & (SUBG - 1)), box_L, box_invL), box_invL);
        const int part = SPLIT ? (int)((kk0 + it) % split) : 0, rounds = SPLIT ? SUBG / split : SUBG;
        for (int q = part * rounds; q < (part + 1) * rounds; ++q) {
            const int u = (warp + q) & (SUBG - 1);
            const BoxShift dec = boxcode_unpack(__shfl_sync(0xffffffffu, my_code, u), box_L);
            if (dec.kind != 0) {                              // else: forces_boxring_kernel evaluates this meeting
                u64 nx[NP], ny[NP], nz[NP], ax[NP], ay[NP], az[NP];
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    nx[p] = pack2(-(float)((double)Xsm[(0 * RI + 2 * p) * THREADS] + dec.s[0]), -(float)((double)Xsm[(0 * RI + 2 * p + 1) * THREADS] + dec.s[0]));
                    ny[p] = pack2(-(float)((double)Xsm[(1 * RI + 2 * p) * THREADS] + dec.s[1]), -(float)((double)Xsm[(1 * RI + 2 * p + 1) * THREADS] + dec.s[1]));
                    nz[p] = pack2(-(float)((double)Xsm[(2 * RI + 2 * p) * THREADS] + dec.s[2]), -(float)((double)Xsm[(2 * RI + 2 * p + 1) * THREADS] + dec.s[2]));
                    ax[p] = ay[p] = az[p] = 0ull;
                }
                for (int t = 0; t < WI / 32; ++t) {
                    const int j0 = u * WI + t * 32;
                    const float* set = cs + (j0 / TJ) * (4 * TJ) + (j0 % TJ);
                    u64 bx = 0ull, by = 0ull, bz = 0ull;
                    switch (dec.mask) {
                        case 0: sym_mixed_box_steps<NP, 0>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        case 1: sym_mixed_box_steps<NP, 1>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        case 2: sym_mixed_box_steps<NP, 2>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        case 3: sym_mixed_box_steps<NP, 3>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        case 4: sym_mixed_box_steps<NP, 4>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        case 5: sym_mixed_box_steps<NP, 5>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        case 6: sym_mixed_box_steps<NP, 6>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                        default: sym_mixed_box_steps<NP, 7>(set, lane, src_lane, nx, ny, nz, m2, ax, ay, az, bx, by, bz, halfL); break;
                    }
                    float lo, hi;
                    const int j = j0 + lane;
                    unpack2(bx, lo, hi); Bsm[j] += (double)lo + (double)hi;
                    unpack2(by, lo, hi); Bsm[IB + j] += (double)lo + (double)hi;
                    unpack2(bz, lo, hi); Bsm[2 * IB + j] += (double)lo + (double)hi;
                    if ((t & 3) == 3) {
#pragma unroll
                        for (int p = 0; p < NP; ++p) {
                            unpack2(ax[p], lo, hi); Asm[(0 * RI + 2 * p) * THREADS] += (double)lo; Asm[(0 * RI + 2 * p + 1) * THREADS] += (double)hi;
                            unpack2(ay[p], lo, hi); Asm[(1 * RI + 2 * p) * THREADS] += (double)lo; Asm[(1 * RI + 2 * p + 1) * THREADS] += (double)hi;
                            unpack2(az[p], lo, hi); Asm[(2 * RI + 2 * p) * THREADS] += (double)lo; Asm[(2 * RI + 2 * p + 1) * THREADS] += (double)hi;
                            ax[p] = ay[p] = az[p] = 0ull;
                        }
                    }
                }
            }
            // (a CTA-wide barrier per round here: the neighbour hand-over of the fp64 kernel, round_wait, measured SLOWER with
            // this kernel's two warps per scheduler -- 30.5 against 28.1 ms at N = 262,144)
            __syncthreads();
        }

        const long long rec = (kk0 + it - k_begin) * 3 * IB;
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            const int i = warp * WI + lane + 32 * k;
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) rowrec[rec + cc * IB + i] = Asm[(cc * RI + k) * THREADS];
        }
        for (int j = threadIdx.x; j < IB; j += THREADS) {
            const double cj = (double)cs[(j / TJ) * (4 * TJ) + 3 * TJ + ((j % TJ) ^ STEPS_C_SWIZZLE)];
            const double f = -cj * cj;
            colrec[rec + j] = f * Bsm[j]; colrec[rec + IB + j] = f * Bsm[IB + j]; colrec[rec + 2 * IB + j] = f * Bsm[2 * IB + j];
        }
        __syncthreads();
        if (threadIdx.x == 0 && it + 2 < total) produce(it + 2);
        if ((kk0 + it + 1) % split == 0 && ++c == nb) { ++b; c = b + 1; }
    }
}

// ---- the pair-symmetric IMAGE SUM (Eq. 5 L65-70 with the 2.6 L cut, second part) ---------------
// The image sum of a pair is antisymmetric like the pair force itself (the image set is symmetric under n -> -n), so every
// far meeting of a warp's 128-particle group with a 128-source subgroup of another block is evaluated ONCE:
// P_ij = sum over the images of (v w), v = (x_j - x_i) - n L, w = |v|^-3 inside the cut, and a_i += m_j P_ij, a_j -= m_i P_ij
// -- one pass over the ~100 candidate images per unordered pair instead of two.  Items, rounds, hand-over of the
// reaction sums round the warp, neighbour hand-over of the subgroups and records as in forces_sym_box_kernel; the
// candidates of a meeting are pruned from the two groups' bounding boxes as in forces_boxring_kernel<Fp64Path, 2> (no
// per-pair wrap: one lattice shift centres the box difference).  A candidate image whose lattice point comes closer to the
// box of separations than the largest pair softening of the two groups MAY be softened: those few (usually none, or the
// one nearest image of neighbouring groups) go through Eq. 4 in full per pair, all others through the branch-free body.
// Only meetings whose boxes span a whole period (pair_too_wide: groups that straddle a jump of the cell order) are skipped
// and evaluated by forces_boxgen_kernel<Fp64Path, 2>, like every group's meeting with itself; the groups' own blocks are
// the diagonal items of this kernel (`diag`).
// The column block arrives as its tiles' PLAIN sources (x, y, z, m, h); the particles' sums live in shared memory.
constexpr int SYM_IMG_NCUBE = 343, SYM_IMG_CAND_STRIDE = 352;
__host__ __device__ constexpr int sym_img_smem_bytes() { return 5 * IB * (int)sizeof(double) + 2 * 3 * IB * (int)sizeof(double); }

template <int THREADS, int RI, bool SPLIT>
__global__ void __launch_bounds__(THREADS, 1)
forces_sym_img_kernel(const TileF64* __restrict__ tiles, const SymPlan* __restrict__ plan, const GroupMeta* __restrict__ gm,
                      long long k_begin, long long k_end, double* __restrict__ rowrec, double* __restrict__ colrec, int split_arg,
                      double box_L, double box_invL, int diag)
{
    // diag != 0: the items are the blocks THEMSELVES, (b, b), b = 0 ... nb - 1: of the two meetings of an unordered pair of
    // groups {w, u} of the block -- warp w with subgroup u, warp u with subgroup w -- the one with (u - w) mod 16 < 8 is
    // evaluated (at distance 8 the one with w < u): every warp has 7 or 8 meetings, each pair of groups is evaluated once.
    // A group's meeting with itself (and whatever pair_too_wide leaves out) is forces_boxgen_kernel's.  Both records of
    // such an item belong to block b (forces_sym_diag_reduce).
    const int split = SPLIT ? split_arg : 1;
    static_assert(THREADS * RI == IB && RI % 2 == 0, "the CTA holds one block; the particles are taken two at a time");
    constexpr int WI = 32 * RI, SUBG = THREADS / 32;
    static_assert(WI == WARP_I && WI * 2 == TJ, "a warp's particles are one group of GroupMeta = half a tile");
    constexpr double A = 1.4;
    constexpr double C0 = 1.0 / STEPS_FP64_FOLD - (1.0 - A) * (1.0 - A);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar;
    __shared__ double cube_tab[3 * SYM_IMG_NCUBE];                                 // offsets n L, n in [-3, 3]^3
    __shared__ unsigned short cand_all[SUBG * SYM_IMG_CAND_STRIDE];                // per warp: the candidates of its meeting
    __shared__ int round_done[SUBG];
    double* col = reinterpret_cast<double*>(smem_raw);                             // [TPB][x, y, z, m, h][TJ]
    double* Bsm = col + 5 * IB;                                                    // [3][IB]
    double* Asm = Bsm + 3 * IB + threadIdx.x;                                      // [3][RI][THREADS], this thread's column
    for (int q = threadIdx.x; q < SYM_IMG_NCUBE; q += THREADS) {
        cube_tab[3 * q] = (double)(q % 7 - 3) * box_L; cube_tab[3 * q + 1] = (double)((q / 7) % 7 - 3) * box_L;
        cube_tab[3 * q + 2] = (double)(q / 49 - 3) * box_L;
    }
    if (threadIdx.x < SUBG) round_done[threadIdx.x] = 0;

    const int nb = plan->nb, Km = plan->Km;     // W = 0: item (b, c) for every c > b
    const long long K = (diag ? (plan->K > 0 ? (long long)nb : 0ll) : plan->K) * split;
    if (k_end > K) k_end = K;
    if (k_begin >= k_end) return;
    const long long n_items = k_end - k_begin;
    const long long kk0 = k_begin + (long long)blockIdx.x * n_items / gridDim.x;
    const long long kk1 = k_begin + ((long long)blockIdx.x + 1) * n_items / gridDim.x;
    const int total = (int)(kk1 - kk0);
    if (total <= 0) return;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int b, c;
    if (diag) {
        b = c = (int)(kk0 / split);
    } else {
        const double t = 2.0 * Km + 1.0;
        const long long item0 = kk0 / split;
        int bb = (int)((t - sqrt(fmax(t * t - 8.0 * (double)item0, 0.0))) * 0.5);
        bb = max(0, min(bb, Km - 1));
        while (bb + 1 < Km && sym_row_start(bb + 1, Km) <= item0) ++bb;
        while (bb > 0 && sym_row_start(bb, Km) > item0) --bb;
        b = bb;
        c = bb + 1 + (int)(item0 - sym_row_start(bb, Km));
    }
    if (threadIdx.x == 0) {
        mbar_init(&full_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int src_lane = (lane + 31) & 31;
    const long long cut2_bits = __double_as_longlong((2.6 * box_L) * (2.6 * box_L));
    const double cut2 = (2.6 * box_L) * (2.6 * box_L), eps = 1.0e-5 * box_L;
    unsigned short* cand = cand_all + warp * SYM_IMG_CAND_STRIDE;

    for (int it = 0; it < total; ++it) {
        // the column block's plain sources: one stage (an item runs for milliseconds; the previous item's readers are past
        // the barrier at its end)
        if (threadIdx.x == 0) {
            mbar_expect_tx(&full_bar, (uint32_t)(5 * IB * sizeof(double)));
#pragma unroll
            for (int t = 0; t < TPB; ++t)
                bulk_load(col + t * 5 * TJ, &tiles[(long long)c * TPB + t].x[0], (uint32_t)(5 * TJ * sizeof(double)), &full_bar);
        }
#pragma unroll
        for (int q = 0; q < 3 * RI; ++q) Asm[q * THREADS] = 0.0;
        for (int q = threadIdx.x; q < 3 * IB; q += THREADS) Bsm[q] = 0.0;
        mbar_wait(&full_bar, it & 1);
        __syncthreads();

        bool my_skip;
        {
            const int uu = lane & (SUBG - 1), dist = (uu - warp) & (SUBG - 1);
            if (diag && (dist == 0 || dist > SUBG / 2 || (dist == SUBG / 2 && warp > uu))) my_skip = true;   // the other meeting's, or the group itself
            else my_skip = pair_too_wide<1>(gm, b * SUBG + warp, c * SUBG + uu, box_L);
        }
        const int part = SPLIT ? (int)((kk0 + it) % split) : 0, rounds = SPLIT ? SUBG / split : SUBG;
        const int base = it * rounds;
        for (int q = part * rounds; q < (part + 1) * rounds; ++q) {
            const int u = (warp + q) & (SUBG - 1);
            if (q > part * rounds) {                          // subgroup u was warp + 1's in the round before (round_wait)
                if (lane == 0) round_wait(&round_done[(warp + 1) & (SUBG - 1)], base + (q - part * rounds));
                __syncwarp();
            }
            if (!__shfl_sync(0xffffffffu, (int)my_skip, u)) {                      // else: forces_boxgen_kernel<., 2> evaluates it
                // the lattice shift that centres the box difference, and the candidates that come within the cut
                const GroupMeta GI = gm[b * SUBG + warp], GJ = gm[c * SUBG + u];
                double sh[3], lo3[3], hi3[3];
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) {
                    const double dmin = ((double)GJ.lo[cc] - (double)GI.hi[cc]) - eps, dmax = ((double)GJ.hi[cc] - (double)GI.lo[cc]) + eps;
                    sh[cc] = box_L * rint(0.5 * (dmin + dmax) * box_invL);
                    lo3[cc] = dmin - sh[cc]; hi3[cc] = dmax - sh[cc];
                }
                // candidates that may be softened go to the back of the list
                const double need = ((double)GI.hmax + (double)GJ.hmax) * 1.0001 + eps, need2 = need * need;
                int ncand = 0, nsoft = 0;
                for (int q0 = 0; q0 < SYM_IMG_NCUBE; q0 += 32) {
                    const int tq = q0 + lane;
                    bool keep = false, softq = false;
                    if (tq < SYM_IMG_NCUBE) {
                        double g2 = 0.0;
#pragma unroll
                        for (int cc = 0; cc < 3; ++cc) {
                            const double o = cube_tab[3 * tq + cc];
                            const double gap = fmax(0.0, fmax(lo3[cc] - o, o - hi3[cc]));
                            g2 = fma(gap, gap, g2);
                        }
                        softq = g2 < cut2 && !(g2 > need2);
                        keep = g2 < cut2 && !softq;
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, keep), ms = __ballot_sync(0xffffffffu, softq);
                    if (keep) cand[ncand + __popc(m & ((1u << lane) - 1u))] = (unsigned short)tq;
                    if (softq) cand[SYM_IMG_CAND_STRIDE - 1 - (nsoft + __popc(ms & ((1u << lane) - 1u)))] = (unsigned short)tq;
                    ncand += __popc(m); nsoft += __popc(ms);
                }
                __syncwarp();
                double xi[RI], yi[RI], zi[RI], mi[RI], hi[RI];
#pragma unroll
                for (int k = 0; k < RI; ++k) {
                    const int i = warp * WI + lane + 32 * k;
                    const TileF64& T = tiles[(long long)b * TPB + i / TJ];
                    xi[k] = T.x[i % TJ] + sh[0]; yi[k] = T.y[i % TJ] + sh[1]; zi[k] = T.z[i % TJ] + sh[2];
                    mi[k] = STEPS_FP64_FOLD * T.m[i % TJ]; hi[k] = T.h[i % TJ];
                }
                for (int t = 0; t < WI / 32 && ncand + nsoft > 0; ++t) {
                    const int s0 = u * WI + t * 32;                                  // first source of the set, within the block
                    double bx = 0.0, by = 0.0, bz = 0.0;
#pragma unroll 1
                    for (int st = 0; st < 32; ++st) {
                        const int s = s0 + ((lane - st) & 31);
                        const double* P = col + (s / TJ) * 5 * TJ + (s % TJ);
                        const double xj = P[0], yj = P[TJ], zj = P[2 * TJ], mq = P[3 * TJ];
                        if (mq != 0.0) {                                         // pads and massless sources add nothing
                            const double mf = STEPS_FP64_FOLD * mq;
#pragma unroll
                            for (int k0 = 0; k0 < RI; k0 += 2) {
                                double dx[2], dy[2], dz[2], px[2], py[2], pz[2];
#pragma unroll
                                for (int k = 0; k < 2; ++k) {
                                    dx[k] = xj - xi[k0 + k]; dy[k] = yj - yi[k0 + k]; dz[k] = zj - zi[k0 + k];
                                    px[k] = py[k] = pz[k] = 0.0;
                                }
                                double nox = 0.0, noy = 0.0, noz = 0.0;
                                if (ncand > 0) { const int t3 = 3 * cand[0]; nox = cube_tab[t3]; noy = cube_tab[t3 + 1]; noz = cube_tab[t3 + 2]; }
#pragma unroll 2
                                for (int cq = 0; cq < ncand; ++cq) {
                                    const double ox = nox, oy = noy, oz = noz;
                                    { const int t3 = 3 * cand[min(cq + 1, ncand - 1)]; nox = cube_tab[t3]; noy = cube_tab[t3 + 1]; noz = cube_tab[t3 + 2]; }
                                    double vx[2], vy[2], vz[2], r2[2], y0[2], y2[2], w[2];
#pragma unroll
                                    for (int k = 0; k < 2; ++k) { vx[k] = dx[k] - ox; vy[k] = dy[k] - oy; vz[k] = dz[k] - oz; }
#pragma unroll
                                    for (int k = 0; k < 2; ++k) r2[k] = fma(vz[k], vz[k], fma(vy[k], vy[k], vx[k] * vx[k]));
#pragma unroll
                                    for (int k = 0; k < 2; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
                                    for (int k = 0; k < 2; ++k) {
                                        y2[k] = y0[k] * y0[k];
                                        w[k] = fma(r2[k], y2[k], -A);
                                        y2[k] = y0[k] * y2[k];
                                        w[k] = fma(w[k], w[k], C0);
                                        w[k] = y2[k] * w[k];
                                        if (!(__double_as_longlong(r2[k]) < cut2_bits)) w[k] = 0.0;   // "|x - nL| < 2.6 L", strict
                                    }
#pragma unroll
                                    for (int k = 0; k < 2; ++k) {
                                        px[k] = fma(vx[k], w[k], px[k]); py[k] = fma(vy[k], w[k], py[k]); pz[k] = fma(vz[k], w[k], pz[k]);
                                    }
                                }
                                if (nsoft > 0) {                                  // the images that may be softened: Eq. 4 in full
                                    const double hj = P[4 * TJ];
#pragma unroll 1
                                    for (int cq = 0; cq < nsoft; ++cq) {
                                        const int t3 = 3 * cand[SYM_IMG_CAND_STRIDE - 1 - cq];
                                        const double ox = cube_tab[t3], oy = cube_tab[t3 + 1], oz = cube_tab[t3 + 2];
#pragma unroll
                                        for (int k = 0; k < 2; ++k) {
                                            const double vx = dx[k] - ox, vy = dy[k] - oy, vz = dz[k] - oz;
                                            const double r2 = fma(vz, vz, fma(vy, vy, vx * vx));
                                            const double hs = hi[k0 + k] + hj;
                                            double sq = Fp64Path::rcube(r2);
                                            if (r2 < hs * hs || r2 == 0.0) sq = (r2 == 0.0) ? 0.0 : spline_g_soft_f64(r2, hs);   // readings #2, #4
                                            if (!(r2 < cut2)) sq = 0.0;
                                            sq *= 1.0 / STEPS_FP64_FOLD;
                                            px[k] = fma(vx, sq, px[k]); py[k] = fma(vy, sq, py[k]); pz[k] = fma(vz, sq, pz[k]);
                                        }
                                    }
                                }
#pragma unroll
                                for (int k = 0; k < 2; ++k) {                     // a_i += m_j P (in shared memory), b_j += m_i P
                                    Asm[(0 * RI + k0 + k) * THREADS] += mf * px[k];
                                    Asm[(1 * RI + k0 + k) * THREADS] += mf * py[k];
                                    Asm[(2 * RI + k0 + k) * THREADS] += mf * pz[k];
                                    bx = fma(mi[k0 + k], px[k], bx); by = fma(mi[k0 + k], py[k], by); bz = fma(mi[k0 + k], pz[k], bz);
                                }
                            }
                        }
                        bx = __shfl_sync(0xffffffffu, bx, src_lane);
                        by = __shfl_sync(0xffffffffu, by, src_lane);
                        bz = __shfl_sync(0xffffffffu, bz, src_lane);
                    }
                    const int j = s0 + lane;
                    Bsm[j] += bx; Bsm[IB + j] += by; Bsm[2 * IB + j] += bz;
                }
            }
            __syncwarp();
            if (lane == 0) round_publish(&round_done[warp], base + (q - part * rounds) + 1);
        }
        __syncthreads();                                      // every subgroup's reaction sums are complete

        const long long rec = (kk0 + it - k_begin) * 3 * IB;
#pragma unroll
        for (int k = 0; k < RI; ++k) {
            const int i = warp * WI + lane + 32 * k;
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) rowrec[rec + cc * IB + i] = Asm[(cc * RI + k) * THREADS];
        }
        for (int j = threadIdx.x; j < IB; j += THREADS) {      // the reaction: a_j -= sum_i m_i P_ij
            colrec[rec + j] = -Bsm[j]; colrec[rec + IB + j] = -Bsm[IB + j]; colrec[rec + 2 * IB + j] = -Bsm[2 * IB + j];
        }
        __syncthreads();                                      // the column stage, Asm and Bsm are free again
        if ((kk0 + it + 1) % split == 0) {
            if (diag) { ++b; c = b; }
            else if (++c == nb) { ++b; c = b + 1; }
        }
    }
}

// The records of the diagonal items of forces_sym_img_kernel (item b, `split` parts: both records are block b's) added to
// the double-double result in fixed order.
__global__ void __launch_bounds__(256)
forces_sym_diag_reduce(const SymPlan* __restrict__ plan, const double* __restrict__ rowrec, const double* __restrict__ colrec, int split,
                       long long N, double* __restrict__ acc_hi, double* __restrict__ acc_lo)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || plan->K <= 0) return;
    const int b = (int)(i / IB), off = (int)(i - (long long)b * IB);
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
        double hi = acc_hi[cc * N + i], lo = acc_lo[cc * N + i];
        for (int p = 0; p < split; ++p) {
            const long long at = ((long long)b * split + p) * 3 * IB + (long long)cc * IB + off;
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const double v = r == 0 ? rowrec[at] : colrec[at];
                const double s = hi + v, bb = s - hi;
                lo += (hi - (s - bb)) + (v - bb);              // TwoSum
                hi = s;
            }
        }
        acc_hi[cc * N + i] = hi; acc_lo[cc * N + i] = lo;
    }
}

// acc (double-double, SoA over all N particles) += the records of one panel, in fixed order; `last` writes acc_out = hi + lo.
__global__ void __launch_bounds__(256)
forces_sym_reduce_kernel(const SymPlan* __restrict__ plan, const double* __restrict__ rowrec, const double* __restrict__ colrec,
                         long long k_begin, long long k_end, long long N, double* __restrict__ acc_hi,
                         double* __restrict__ acc_lo, int last, double* __restrict__ acc_out, int split, Eq12Fuse fuse,
                         int share_rank = 0, int share_world = 1)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double dt = __longlong_as_double((long long)STEPS_DT_INF_BITS);
    if (i < N) {
    const long long Kall = plan->K * split;            // sub-items (see forces_sym_kernel); the rank's share of them
    const long long S0 = Kall * share_rank / share_world, K = Kall * (share_rank + 1) / share_world;
    k_begin += S0; k_end += S0;
    if (k_end > K) k_end = K;
    const int Km = plan->Km, pnb = plan->nb;
    const long long* rowstart = plan_rowstart(plan, pnb);
    const int* edge = plan_edge(plan, pnb);
    const int b = (int)(i / IB), off = (int)(i - (long long)b * IB);
    double hi[3], lo[3];
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) { hi[cc] = acc_hi[cc * N + i]; lo[cc] = acc_lo[cc * N + i]; }
    auto add = [&](const double* rec, long long k) {
        const double* p = rec + (k - k_begin) * 3 * IB + off;
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            const double v = p[(long long)cc * IB];
            const double s = hi[cc] + v, bb = s - hi[cc];
            lo[cc] += (hi[cc] - (s - bb)) + (v - bb);              // TwoSum
            hi[cc] = s;
        }
    };
    if (k_begin < k_end) {
        if (b < Km) {                                              // this block as the row of its items
            const long long r0 = rowstart[b] * split, r1 = rowstart[b + 1] * split;
            for (long long k = max(r0, k_begin); k < min(r1, k_end); ++k) add(rowrec, k);
        }
        // this block as the column of item (bb, b): the rows bb with edge[bb] < b, i.e. bb < lo[b]; of those, the rows
        // that have items inside [k_begin, k_end)
        const int rows = min(Km, plan_lo(plan, pnb)[b]);
        const int bb_first = sym_row_of(rowstart, Km, k_begin / split), bb_last = sym_row_of(rowstart, Km, (k_end - 1) / split);
        for (int bb = bb_first; bb < min(rows, bb_last + 1); ++bb) {
            const long long k0 = (rowstart[bb] + (b - edge[bb] - 1)) * split;
            for (long long k = max(k0, k_begin); k < min(k0 + split, k_end); ++k) add(colrec, k);
        }
    }
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
        if (last) acc_out[cc * N + i] = hi[cc] + lo[cc];
        else { acc_hi[cc * N + i] = hi[cc]; acc_lo[cc * N + i] = lo[cc]; }
    }
    if (last && fuse.out_bits) {
        const double a = *fuse.a_state, coef = fuse.absG / (a * a * a);
        dt = eq12_candidate(hi[0] + lo[0], hi[1] + lo[1], hi[2] + lo[2], fuse.pos[i], fuse.pos[N + i], fuse.pos[2 * N + i], fuse.soft[i],
                            coef, fuse.B, fuse.eps, dt);
    }
    }
    if (last && fuse.out_bits) eq12_fold(fuse, dt);
}

}  // namespace steps
