// force_driver.cuh -- the two force drivers that move j-tiles past register-blocked i-particles.
//
//  forces_persistent_kernel  (default): persistent CTAs (grid = SMs x resident CTAs), the
//      (i-block, j-tile) iteration space is linearised and cut into equal contiguous shares
//      ("stream-K"), so every CTA streams the same number of tiles no matter how N divides.
//      j-tiles arrive in shared memory by 1-D bulk TMA copies (cp.async.bulk -> UBLKCP in SASS)
//      through a STAGES-deep mbarrier ring; one elected thread is the producer.  A CTA whose
//      share crosses an i-block boundary writes one partial record per i-block it touched;
//      forces_reduce_kernel sums the records of each i-block in fixed CTA order (deterministic).
//  forces_v1_kernel: one CTA per i-block, plain loads + __syncthreads.  Kept as the in-library
//      cross-check of the persistent driver (steps_set_option("driver", 1)).
//
// `zero` is a kernel argument that is always 0 and that the compiler cannot know to be 0: the fp64 far
// body tests bits of it to place never-taken branches between its stages (see force_fp64.cuh).
//
// Both share the Path bodies (force_mixed.cuh / force_fp64.cuh) and the per-thread accumulator
// block in shared memory: element (c, k) of thread t at acc[(c * R_I + k) * CTA_THREADS + t].
#pragma once
#include "common.cuh"
#include "force_fp64.cuh"   // EWALD_NTRIPLETS / ewald_triplets (image-sum table of BOX = 2)

namespace steps {

// ---- mbarrier / bulk-copy PTX ------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LAB_DONE;\n"
        "bra LAB_WAIT;\n"
        "LAB_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared, completion signalled on an mbarrier (TMA engine, no tensor map).
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---- shared helpers ----------------------------------------------------------------------------
template <typename Path>
__device__ __forceinline__ void load_i_block(typename Path::IState& S, const double* __restrict__ pos,
                                             const double* __restrict__ soft, long long N, long long i0,
                                             long long i_end, float& rlo, float& rhi, float& hh)
{
    long long idx[R_I];
#pragma unroll
    for (int k = 0; k < R_I; ++k) {
        const long long i = i0 + 32 * k;
        idx[k] = i < i_end ? i : i_end - 1;     // clamp: duplicates a real particle, result not stored
    }
    rlo = __int_as_float(0x7f800000); rhi = 0.0f; hh = 0.0f;
    Path::load_i(S, pos, soft, N, idx, rlo, rhi, hh);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {          // bounds of the warp's 128 contiguous i-particles
        rlo = fminf(rlo, __shfl_xor_sync(0xffffffffu, rlo, o));
        rhi = fmaxf(rhi, __shfl_xor_sync(0xffffffffu, rhi, o));
        hh = fmaxf(hh, __shfl_xor_sync(0xffffffffu, hh, o));
    }
}

// Bounding box of the warp's 128 i-particles, rounded outwards (periodic boxes: box_shift in common.cuh).
template <typename Path>
__device__ __forceinline__ void warp_box(const typename Path::IState& S, float (&lo)[3], float (&hi)[3])
{
    const float inf = __int_as_float(0x7f800000);
#pragma unroll
    for (int c = 0; c < 3; ++c) { lo[c] = inf; hi[c] = -inf; }
#pragma unroll
    for (int k = 0; k < R_I; ++k) {
        const double v[3] = {(double)S.x[k], (double)S.y[k], (double)S.z[k]};
#pragma unroll
        for (int c = 0; c < 3; ++c) { lo[c] = fminf(lo[c], __double2float_rd(v[c])); hi[c] = fmaxf(hi[c], __double2float_ru(v[c])); }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o));
            hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
        }
}

// FarSums of the fp64 path are register sums (zeroed); those of the mixed path only carry the accumulator pointer.
template <typename Path>
__device__ __forceinline__ void init_far_sums(typename Path::FarSums& F, double* acc)
{
    if constexpr (Path::NOUT == 3) F.acc = acc;
    else Path::far_zero(F);
}

// Periodic far body of a (group, tile) pair; Q = the group with the pair's image shift on it, the fold mask picks the body.
template <typename Path>
__device__ __forceinline__ void far_fold_dispatch(const typename Path::Tile& T, const typename Path::IState& Q, typename Path::FarSums& F,
                                                  int zero, int mask, double halfL, int j0, int j1)
{
    switch (mask) {
        case 0: Path::template far_fold<0>(T, Q, F, zero, halfL, j0, j1); break;
        case 1: Path::template far_fold<1>(T, Q, F, zero, halfL, j0, j1); break;
        case 2: Path::template far_fold<2>(T, Q, F, zero, halfL, j0, j1); break;
        case 3: Path::template far_fold<3>(T, Q, F, zero, halfL, j0, j1); break;
        case 4: Path::template far_fold<4>(T, Q, F, zero, halfL, j0, j1); break;
        case 5: Path::template far_fold<5>(T, Q, F, zero, halfL, j0, j1); break;
        case 6: Path::template far_fold<6>(T, Q, F, zero, halfL, j0, j1); break;
        default: Path::template far_fold<7>(T, Q, F, zero, halfL, j0, j1); break;
    }
}

// The decision of box_shift packed into one word (forces_boxring_kernel keeps one per tile in shared memory):
// bits 0-2 fold mask, bit 3 general body, bits 8-15 / 16-23 / 24-31 the shifts in units of L/2 (signed bytes).
constexpr uint32_t BOXCODE_GENERAL = 8u;
__device__ __forceinline__ uint32_t boxcode_pack(const BoxShift& bs, double invL)
{
    if (bs.kind == 0) return BOXCODE_GENERAL;
    uint32_t code = (uint32_t)bs.mask;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double k2 = rint(2.0 * bs.s[c] * invL);           // an integer by construction (k L or (k + 1/2) L)
        if (!(fabs(k2) <= 127.0)) return BOXCODE_GENERAL;       // particles many periods apart: the general body wraps them
        code |= ((uint32_t)(int)k2 & 0xffu) << (8 + 8 * c);
    }
    return code;
}
__device__ __forceinline__ BoxShift boxcode_unpack(uint32_t code, double L)
{
    BoxShift bs;
    bs.kind = (code & BOXCODE_GENERAL) ? 0 : 1;
    bs.mask = (int)(code & 7u);
#pragma unroll
    for (int c = 0; c < 3; ++c) bs.s[c] = (double)(int)(signed char)((code >> (8 + 8 * c)) & 0xffu) * (0.5 * L);   // exact: see box_shift
    return bs;
}

__host__ __device__ constexpr int stage_stride(int tile_bytes) { return (tile_bytes + 127) / 128 * 128; }

template <typename Path, int STAGES>
constexpr int persistent_smem_bytes()
{
    return STAGES * stage_stride((int)sizeof(typename Path::Tile)) + Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double);
}

// ---- band mode (force_sym.cuh) ---------------------------------------------------------------------
// Device-resident plan of a pair-symmetric force evaluation (written by sym_band_width + sym_plan_finalize in force_sym.cuh).
// Row b's band is the blocks lo[b] ... edge[b]: edge[b] >= b is the last block that is not provably far from b or from an
// earlier row (made non-decreasing in b, so that the band is symmetric: c <= edge[b]  <=>  b >= lo[c] for b <= c), and
// lo[c] = the first row whose edge reaches c.  In BAND mode the persistent driver only visits, for i-block b, the tiles of
// its band; the block pairs (b, c) with c > edge[b] are the work items of forces_sym_kernel, row after row.
struct SymPlan {
    int W;            // widest band: max (edge[b] - b); nb - 1 = no symmetric items
    int nb;           // blocks
    int Km;           // rows that own symmetric items (rows 0 ... Km - 1: edge[b] < nb - 1)
    int nt;           // j-tiles, padded to whole blocks: nb * (IB / TJ)
    long long K;      // symmetric items: rowstart[nb]
    long long T;      // band tile visits: cum[nb]
};
// followed in memory by  long long cum[nb + 1]: band tile visits of the rows before b,
//                        long long rowstart[nb + 1]: symmetric items of the rows before b,  int edge[nb],  int lo[nb]
__host__ __device__ inline size_t sym_plan_bytes(long long nb)
{
    return sizeof(SymPlan) + 2 * sizeof(long long) * (size_t)(nb + 1) + 2 * sizeof(int) * (size_t)nb;
}
__device__ __forceinline__ const long long* plan_cum(const SymPlan* plan) { return reinterpret_cast<const long long*>(plan + 1); }
__device__ __forceinline__ const long long* plan_rowstart(const SymPlan* plan, int nb) { return plan_cum(plan) + nb + 1; }
__device__ __forceinline__ const int* plan_edge(const SymPlan* plan, int nb) { return reinterpret_cast<const int*>(plan_rowstart(plan, nb) + nb + 1); }
__device__ __forceinline__ const int* plan_lo(const SymPlan* plan, int nb) { return plan_edge(plan, nb) + nb; }
// the row of symmetric item k: the largest b < Km with rowstart[b] <= k
__device__ __forceinline__ int sym_row_of(const long long* __restrict__ rowstart, int Km, long long k)
{
    int lo = 0, hi = max(Km - 1, 0);
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (rowstart[mid] <= k) lo = mid; else hi = mid - 1;
    }
    return lo;
}
// row b of the band with cum[b] <= w < cum[b + 1]
__device__ __forceinline__ int band_row_of(const long long* __restrict__ cum, int nb, long long w)
{
    int lo = 0, hi = nb - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (cum[mid] <= w) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// The item list of the symmetric kernels (kept out of line: the kernels' register allocation is tuned to the body, and the
// lookups run once per CTA / once per row).  Item k is the block pair (b, c): b = its row, c = edge[b] + 1 + (k - rowstart[b]).
__device__ __noinline__ int2 sym_item_decode(const SymPlan* plan, long long k)
{
    const int nb = plan->nb;
    const long long* rowstart = plan_rowstart(plan, nb);
    const int b = sym_row_of(rowstart, plan->Km, k);
    return make_int2(b, plan_edge(plan, nb)[b] + 1 + (int)(k - rowstart[b]));
}
// the column of the first item of row b
__device__ __noinline__ int sym_row_first_col(const SymPlan* plan, int b)
{
    const int nb = plan->nb;
    return plan_edge(plan, nb)[min(b, nb - 1)] + 1;
}

// ---- persistent stream-K driver ------------------------------------------------------------------
// partials: [nb + gridDim.x slots][Path::NOUT][IB] doubles; CTA p's record for i-block b is slot b + p.
// (Periodic boxes, have their own driver: forces_boxring_kernel below.  BOX stays a parameter of the
// launchers; here it is always 0.)
// BAND (open boundary only): the iteration space is the band of `plan` instead of all nb x nt (i-block, tile) pairs.
template <typename Path, int STAGES, int BOX = 0, bool BAND = false>
__global__ void __launch_bounds__(CTA_THREADS, 1)
forces_persistent_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                         const typename Path::Tile* __restrict__ tiles, int nt, long long i_begin, long long i_end,
                         int nb, double* __restrict__ partials, int zero, double box_L, double box_invL,
                         const SymPlan* __restrict__ plan, int block_stride, int share_rank = 0, int share_world = 1)
{
    // BAND mode, share_world > 1 (steps_forces_share): only the share_rank-th of share_world equal parts of the band's
    // (i-block, tile) visits; forces_band_reduce_kernel gets the same two numbers.
    // block_stride > 1 (multi-GPU dealing, steps_forces_blocks): local i-block b is the global block
    // i_begin / IB + b * block_stride; i_end is then N.
    static_assert(!BAND || BOX == 0, "the band split applies to the open boundary only");
    static_assert(BOX == 0, "periodic boxes run on forces_boxring_kernel");
    using Tile = typename Path::Tile;
    constexpr int STRIDE = stage_stride((int)sizeof(Tile));
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[STAGES], empty_bar[STAGES];
    double* acc = reinterpret_cast<double*>(smem_raw + STAGES * STRIDE) + threadIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long* cum = BAND ? plan_cum(plan) : nullptr;
    const long long Wall = BAND ? plan->T : (long long)nb * nt;
    const long long R0 = BAND ? Wall * share_rank / share_world : 0, R1 = BAND ? Wall * (share_rank + 1) / share_world : Wall;
    const long long W = R1 - R0;
    const long long w0 = R0 + (long long)blockIdx.x * W / gridDim.x;
    const long long w1 = R0 + ((long long)blockIdx.x + 1) * W / gridDim.x;
    const int total = (int)(w1 - w0);                       // tiles this CTA streams
    if (total <= 0) return;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], CTA_THREADS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // producer (thread 0): tile number k of this CTA's stream is tiles[(w0 + k) % nt], stage k % STAGES
    auto produce = [&](int k) {
        const int s = k % STAGES;
        if (k >= STAGES) mbar_wait(&empty_bar[s], ((k / STAGES) - 1) & 1);
        mbar_expect_tx(&full_bar[s], (uint32_t)sizeof(Tile));
        long long tile;
        if constexpr (BAND) {                                   // band mode: row of the linear index, then its tile
            const int pb = band_row_of(cum, nb, w0 + k);
            tile = (long long)plan_lo(plan, nb)[pb] * (IB / TJ) + (w0 + k - cum[pb]);
        } else {
            tile = (w0 + k) % nt;
        }
        bulk_load(smem_raw + s * STRIDE, tiles + tile, (uint32_t)sizeof(Tile), &full_bar[s]);
    };
    if (threadIdx.x == 0) {
        for (int k = 0; k < STAGES - 1 && k < total; ++k) produce(k);
    }

    int it = 0;                                             // tiles consumed so far
    long long w = w0;
    while (w < w1) {
        int b, cnt;
        if constexpr (BAND) {
            b = band_row_of(cum, nb, w);
            cnt = (int)min(cum[b + 1] - w, w1 - w);
        } else {
            b = (int)(w / nt);
            const int t0 = (int)(w - (long long)b * nt);
            cnt = (int)min((long long)(nt - t0), w1 - w);
        }

        typename Path::IState S;
        float rlo, rhi, hh;
        const long long i0 = i_begin + (long long)b * block_stride * IB + warp * WARP_I + lane;
        load_i_block<Path>(S, pos, soft, N, i0, i_end, rlo, rhi, hh);
#pragma unroll
        for (int q = 0; q < Path::NOUT * R_I; ++q) acc[q * CTA_THREADS] = 0.0;

        typename Path::FarSums F;
        init_far_sums<Path>(F, acc);
        int pending = 0;                                    // far tiles summed in F since its last flush
        for (int c = 0; c < cnt; ++c, ++it) {
            if (threadIdx.x == 0 && it + STAGES - 1 < total) produce(it + STAGES - 1);
            const int s = it % STAGES;
            mbar_wait(&full_bar[s], (it / STAGES) & 1);
            const Tile& T = *reinterpret_cast<const Tile*>(smem_raw + s * STRIDE);
            {
            // the decision is warp-uniform by construction (warp-reduced bounds); the vote tells the compiler so
            if (__all_sync(0xffffffffu, tile_is_far(rlo, rhi, hh, T.meta))) {
                Path::far(T, S, F, zero);
                if (++pending >= Path::FAR_TILES_PER_FLUSH) { Path::far_flush(F, acc); pending = 0; }
            } else {
                if (pending) { Path::far_flush(F, acc); pending = 0; }
                Path::near(T, S, acc);
            }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[s]);
        }

        if (pending) Path::far_flush(F, acc);
        double* out = partials + ((long long)(b + blockIdx.x) * Path::NOUT) * IB + warp * WARP_I + lane;
#pragma unroll
        for (int cc = 0; cc < Path::NOUT; ++cc)
#pragma unroll
            for (int k = 0; k < R_I; ++k) out[(long long)cc * IB + 32 * k] = acc[(cc * R_I + k) * CTA_THREADS];
        w += cnt;
    }
}

// Fixed-order sum of the partial records of each i-block -> acc_out (SoA over [i_begin, i_end)).
template <int NOUT>
__global__ void __launch_bounds__(256) forces_reduce_kernel(const double* __restrict__ partials, int nt, int nb, int P,
                                                            long long cnt, double* __restrict__ acc_out, Eq12Fuse fuse)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double dt = __longlong_as_double((long long)STEPS_DT_INF_BITS);
    if (i < cnt) {
    double a3[3];
    const int b = (int)(i / IB), off = (int)(i - (long long)b * IB);
    const long long W = (long long)nb * nt;
    // CTA p owns w in [floor(p W / P), floor((p+1) W / P));  the CTA that owns w is floor(((w+1) P - 1) / W)
    const int p_lo = (int)((((long long)b * nt + 1) * P - 1) / W);
    const int p_hi = (int)((((long long)(b + 1) * nt) * P - 1) / W);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double hi = 0.0, lo = 0.0;
        for (int p = p_lo; p <= p_hi; ++p) {
            const long long w0 = (long long)p * W / P, w1 = ((long long)p + 1) * W / P;
            if (w1 <= w0) continue;                                    // idle CTA wrote nothing
            const double* rec = partials + ((long long)(b + p) * NOUT) * IB + off;
            const double v = rec[(long long)c * IB];
            const double s = hi + v, bb = s - hi;
            lo += (hi - (s - bb)) + (v - bb);                          // TwoSum
            hi = s;
            if (NOUT == 6) lo += rec[(long long)(3 + c) * IB];
        }
        a3[c] = hi + lo;
        acc_out[(long long)c * cnt + i] = a3[c];
    }
    if (fuse.out_bits) {                                    // full evaluations only: i is the particle index, cnt = N
        const double a = *fuse.a_state, coef = fuse.absG / (a * a * a);
        dt = eq12_candidate(a3[0], a3[1], a3[2], fuse.pos[i], fuse.pos[cnt + i], fuse.pos[2 * cnt + i], fuse.soft[i], coef, fuse.B,
                            fuse.eps, dt);
    }
    }
    if (fuse.out_bits) eq12_fold(fuse, dt);                 // all 32 lanes of every warp, valid particle or not
}

// The same for the BAND mode (rows of different lengths: the owners of a row come from the plan's cumulative counts).
// to_dd != 0: the result stays double-double in (acc_hi, acc_lo) for forces_sym_reduce_kernel to add its records to.
template <int NOUT>
__global__ void __launch_bounds__(256) forces_band_reduce_kernel(const double* __restrict__ partials, const SymPlan* __restrict__ plan,
                                                                 int P, long long cnt, double* __restrict__ acc_out,
                                                                 int to_dd, double* __restrict__ acc_hi, double* __restrict__ acc_lo,
                                                                 int share_rank = 0, int share_world = 1)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cnt) return;
    const long long* cum = plan_cum(plan);
    // the share [R0, R1) of the band's visits that the kernel ran; CTA p owns the local visits [floor(p W / P), floor((p+1) W / P))
    const long long R0 = plan->T * share_rank / share_world, R1 = plan->T * (share_rank + 1) / share_world;
    const long long W = R1 - R0;
    const int b = (int)(i / IB), off = (int)(i - (long long)b * IB);
    const long long v0 = max(cum[b], R0) - R0, v1 = min(cum[b + 1], R1) - R0;      // this block's visits inside the share
    const int p_lo = v0 < v1 ? (int)(((v0 + 1) * P - 1) / W) : 1;
    const int p_hi = v0 < v1 ? (int)((v1 * P - 1) / W) : 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double hi = 0.0, lo = 0.0;
        for (int p = p_lo; p <= p_hi; ++p) {
            const long long w0 = (long long)p * W / P, w1 = ((long long)p + 1) * W / P;
            if (w1 <= w0) continue;
            const double* rec = partials + ((long long)(b + p) * NOUT) * IB + off;
            const double v = rec[(long long)c * IB];
            const double s = hi + v, bb = s - hi;
            lo += (hi - (s - bb)) + (v - bb);                          // TwoSum
            hi = s;
            if (NOUT == 6) lo += rec[(long long)(3 + c) * IB];
        }
        if (to_dd) { acc_hi[(long long)c * cnt + i] = hi; acc_lo[(long long)c * cnt + i] = lo; }
        else acc_out[(long long)c * cnt + i] = hi + lo;
    }
}

// ---- split-j driver ------------------------------------------------------------------------------------------------
// One i-GROUP of 128 particles (4 per lane) per CTA column, the j-range SPLIT over the 16 warps of the CTA (and over
// gridDim.y CTAs): every warp holds the same 128 particles and sums its own work units -- (tile, range of `sub` sources)
// pairs, unit u of the CTA going to warp u mod 16 -- straight from the tile records in global memory (L1/L2: a warp reads
// one record at a time for all its lanes).  The warps' partial accelerations meet in shared memory and are added in fixed
// warp order (TwoSum, double-double): row a3 of the hot path as north_star words it, "reduction of split-j partial
// accelerations", deterministic.  Used where the ring driver's 2,048-particle i-blocks are too coarse:
//   * small N (open boundary): N = 4,096 is 2 i-blocks x 16 tiles for 148 SMs in the ring driver; here 32 groups x 64 units;
//   * periodic boxes (BOX = 1): the far/near/shift decision is per (warp's group, tile) and its cost varies by 2x; warps
//     that share a tile ring wait for the slowest of them at every tile, warps with their own units do not.
// gridDim = (groups, jsplit); partials (jsplit > 1): [group][jsplit][3 or 6][128] doubles, summed by forces_splitj_reduce.
constexpr int SPLITJ_GROUP = WARP_I;                       // 128 i-particles per CTA

template <typename Path, int BOX>
__global__ void __launch_bounds__(CTA_THREADS, 1)
forces_splitj_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                     const typename Path::Tile* __restrict__ tiles, int nt, int sub, long long i_begin, long long i_end,
                     double* __restrict__ acc_out, double* __restrict__ partials, int zero, double box_L, double box_invL,
                     Eq12Fuse fuse, const SymPlan* __restrict__ plan, double* __restrict__ acc_lo_out)
{
    // plan != nullptr: BAND mode of a pair-symmetric evaluation with few blocks (the ring driver's (i-block, tile) items are
    // then too few for 148 SMs: N = 32,768 is 384 visits): the group only meets the tiles of the blocks within the plan's
    // band half-width of its own block, and the result stays double-double (acc_out = hi, acc_lo_out = lo).
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double res[3][SPLITJ_GROUP];                                // the group's final accelerations (Eq. 12 fusion)
    double* acc_all = reinterpret_cast<double*>(smem_raw);                 // [NOUT * R_I][CTA_THREADS]
    double* acc = acc_all + threadIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long cnt = i_end - i_begin;
    typename Path::IState S;
    float rlo, rhi, hh;
    const long long i0 = i_begin + (long long)blockIdx.x * SPLITJ_GROUP + lane;      // the same particles in every warp
    load_i_block<Path>(S, pos, soft, N, i0, i_end, rlo, rhi, hh);
    static_assert(BOX == 0, "periodic boxes run on forces_boxring_kernel / the persistent driver");
#pragma unroll
    for (int q = 0; q < Path::NOUT * R_I; ++q) acc[q * CTA_THREADS] = 0.0;

    const int per_tile = TJ / sub;
    int t_lo = 0, t_hi = nt;                                                // the tiles this group meets
    if (plan != nullptr) {
        const int b = (int)(((long long)blockIdx.x * SPLITJ_GROUP) / IB), pnb = plan->nb;
        t_lo = plan_lo(plan, pnb)[b] * (IB / TJ);
        t_hi = min(nt, (plan_edge(plan, pnb)[b] + 1) * (IB / TJ));
    }
    const long long units = (long long)(t_hi - t_lo) * per_tile;
    const long long u0 = (long long)blockIdx.y * units / gridDim.y, u1 = ((long long)blockIdx.y + 1) * units / gridDim.y;
    typename Path::FarSums F;
    init_far_sums<Path>(F, acc);
    int pending = 0;
    for (long long u = u0 + warp; u < u1; u += CTA_THREADS / 32) {
        const typename Path::Tile& T = tiles[t_lo + u / per_tile];
        const int j0 = (int)(u % per_tile) * sub, j1 = j0 + sub;
        const TileMeta meta = T.meta;
        {
            if (__all_sync(0xffffffffu, tile_is_far(rlo, rhi, hh, meta))) {
                Path::template far<true>(T, S, F, zero, j0, j1);
                if (++pending >= Path::FAR_TILES_PER_FLUSH) { Path::far_flush(F, acc); pending = 0; }
            } else {
                if (pending) { Path::far_flush(F, acc); pending = 0; }
                Path::near(T, S, acc, j0, j1);
            }
        }
    }
    if (pending) Path::far_flush(F, acc);
    __syncthreads();

    // fixed-order sum over the 16 warps: thread (c, k, l) owns component c of particle l + 32 k of the group
    if (threadIdx.x < 3 * SPLITJ_GROUP) {
        const int c = threadIdx.x / SPLITJ_GROUP, r = threadIdx.x % SPLITJ_GROUP, k = r / 32, l = r % 32;
        double hi = 0.0, lo = 0.0;
        for (int w = 0; w < CTA_THREADS / 32; ++w) {
            const double v = acc_all[(c * R_I + k) * CTA_THREADS + w * 32 + l];
            const double s = hi + v, bb = s - hi;
            lo += (hi - (s - bb)) + (v - bb);                              // TwoSum
            hi = s;
            if (Path::NOUT == 6) lo += acc_all[((3 + c) * R_I + k) * CTA_THREADS + w * 32 + l];
        }
        const long long i = (long long)blockIdx.x * SPLITJ_GROUP + l + 32 * k;        // within [i_begin, i_end)
        if (gridDim.y == 1) {
            if (i < cnt) {
                if (acc_lo_out) { acc_out[(long long)c * cnt + i] = hi; acc_lo_out[(long long)c * cnt + i] = lo; }
                else acc_out[(long long)c * cnt + i] = hi + lo;
            }
            res[c][r] = hi + lo;
        } else {
            double* rec = partials + (((long long)blockIdx.x * gridDim.y + blockIdx.y) * 6) * SPLITJ_GROUP;
            rec[c * SPLITJ_GROUP + r] = hi; rec[(3 + c) * SPLITJ_GROUP + r] = lo;
        }
    }
    if (fuse.out_bits != nullptr && gridDim.y == 1) {                       // full evaluations only (i_begin = 0, cnt = N)
        __syncthreads();
        if (threadIdx.x < SPLITJ_GROUP) {
            const int r = threadIdx.x, k = r / 32, l = r % 32;
            const long long i = (long long)blockIdx.x * SPLITJ_GROUP + l + 32 * k;
            double dt = __longlong_as_double((long long)STEPS_DT_INF_BITS);
            if (i < cnt) {
                const double a = *fuse.a_state, coef = fuse.absG / (a * a * a);
                dt = eq12_candidate(res[0][r], res[1][r], res[2][r], fuse.pos[i], fuse.pos[cnt + i], fuse.pos[2 * cnt + i], fuse.soft[i],
                                    coef, fuse.B, fuse.eps, dt);
            }
            eq12_fold(fuse, dt);
        }
    }
}

// acc_lo_out != nullptr: the result stays double-double (acc_out = hi, acc_lo_out = lo) for forces_sym_reduce_kernel.
__global__ void __launch_bounds__(128) forces_splitj_reduce(const double* __restrict__ partials, int jsplit, long long cnt,
                                                            double* __restrict__ acc_out, Eq12Fuse fuse,
                                                            double* __restrict__ acc_lo_out = nullptr)
{
    const int r = threadIdx.x, k = r / 32, l = r % 32;
    const long long i = (long long)blockIdx.x * SPLITJ_GROUP + l + 32 * k;
    double dt = __longlong_as_double((long long)STEPS_DT_INF_BITS);
    if (i < cnt) {
    double a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double hi = 0.0, lo = 0.0;
        for (int s = 0; s < jsplit; ++s) {
            const double* rec = partials + (((long long)blockIdx.x * jsplit + s) * 6) * SPLITJ_GROUP;
            const double v = rec[c * SPLITJ_GROUP + r];
            const double t = hi + v, bb = t - hi;
            lo += (hi - (t - bb)) + (v - bb);
            hi = t;
            lo += rec[(3 + c) * SPLITJ_GROUP + r];
        }
        a3[c] = hi + lo;
        if (acc_lo_out) { acc_out[(long long)c * cnt + i] = hi; acc_lo_out[(long long)c * cnt + i] = lo; }
        else acc_out[(long long)c * cnt + i] = a3[c];
    }
    if (fuse.out_bits) {
        const double a = *fuse.a_state, coef = fuse.absG / (a * a * a);
        dt = eq12_candidate(a3[0], a3[1], a3[2], fuse.pos[i], fuse.pos[cnt + i], fuse.pos[2 * cnt + i], fuse.soft[i], coef, fuse.B,
                            fuse.eps, dt);
    }
    }
    if (fuse.out_bits) eq12_fold(fuse, dt);
}

// ---- group-ring driver: periodic boxes (Eq. 5); BOX = 1 leading image, 2 image sum --------
// One i-GROUP of 128 particles (4 per lane) per CTA column, held by ALL 16 warps of the CTA.  The warps form BOXRING_G
// sub-rings of 4 warps; each sub-ring streams every fourth tile of the range through its own bulk-copy ring (its first
// lane is the producer) and each of its warps takes a quarter (64 sources) of every tile.
// Why this shape: in a periodic box the image decision (box_shift: far or possibly softened, the shift, which components
// fold) is per (group, tile) pair and its cost differs by up to 2x.  Warps that hold DIFFERENT groups and share a tile
// ring wait for the slowest decision at every tile; warps that hold the SAME group all run the same body on a tile, so a
// ring stays in step and every load is a shared-memory broadcast.  The decisions -- one word per tile -- are computed by
// the whole CTA ahead of the rings, DEC_CHUNK tiles at a time, so they cost nothing in the loop, and the producers know
// them: only the FAR part of a tile record (the scaled sources, 8 KiB fp64 / 4 KiB fp32) is copied, and only for tiles
// that take the far body; the rare tile that may hold a softened pair is read by the general wrapped body straight from
// global memory.
// The 16 partial accelerations meet in shared memory and are added in fixed warp order (TwoSum), as in the split-j
// driver; gridDim.y > 1 splits the tile range over CTAs (records summed by forces_splitj_reduce).
// RESTRICTED mode (plan != nullptr and the plan kept its items, W < nb - 1): the pairs of two DIFFERENT blocks of 2,048
// particles belong to the pair-symmetric kernel (forces_sym_box_kernel, force_sym.cuh) and to forces_boxgen_kernel below
// (the units that may hold a softened pair); this kernel then evaluates the group's own block only and ADDS its result to
// the double-double (acc_out = hi, acc_lo_out = lo) that forces_boxgen_kernel wrote.
// BOX = 2: the image sum of Eq. 5 with the 2.6 L cut (fp64) on the same driver.  A far (group, tile) pair -- no image of
// any of its pairs can be softened -- has its candidate images PRUNED from the two bounding boxes: with the lattice shift
// that centres the box difference every separation of the pair lies in [a, b] per component, and image n can come
// within the cut only if the distance from n L to that box is below 2.6 L (about 90-110 of the 343 n in [-3, 3]^3 for
// compact cells; a pair on its own needs 179).  The ring then carries the tile's PLAIN sources; the other tiles go
// through Fp64Path::near_images from global memory.  All warps of the CTA hold the same group, so they all have the same
// candidate list for a tile (each warp builds its own copy) and the same cost: warps holding different groups would wait
// at every tile for the one whose pair is not far (179 candidates + the softening tests).
constexpr int BOXRING_G = 4;                               // sub-rings per CTA
constexpr int DEC_CHUNK = 512;                             // decisions per sub-ring kept in shared memory at a time
template <typename Path, int BOX>
__host__ __device__ constexpr int boxring_stages() { return BOX == 2 ? 2 : 3; }     // stages per sub-ring
template <typename Path, int BOX>
__host__ __device__ constexpr int boxring_part_bytes()     // what the ring carries of a tile record (common.cuh)
{
    // BOX = 1: the scaled sources, which lead the record; BOX = 2: the plain sources x[], y[], z[], m[], h[] that follow them
    return BOX == 2 ? 5 * TJ * (int)sizeof(double) : (Path::NOUT == 6 ? TJ * (int)sizeof(FarSrcF64) : 4 * TJ * (int)sizeof(float));
}
template <typename Path, int BOX>
constexpr int boxring_smem_bytes()
{
    return BOXRING_G * boxring_stages<Path, BOX>() * boxring_part_bytes<Path, BOX>() +
           Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double) + BOXRING_G * DEC_CHUNK * (int)sizeof(uint32_t);
}

// The general body of the group-ring driver as a CALL: it is the rare path (a tile that may hold a softened pair), and
// inlined next to the far loops it costs them registers -- ptxas then spills the i-particles inside the far loop (measured:
// 12 local loads per source).  The group's particles come from the shared-memory copy `gs` ([x, y, z, h][R_I][32 lanes]).
template <typename Path, int BOX>
__device__ __noinline__ void boxring_general(const typename Path::Tile* __restrict__ T, const void* __restrict__ gs_raw, double* acc,
                                             double L, double invL, const double* __restrict__ img_tab, int j0, int j1)
{
    using IState = typename Path::IState;
    using Elem = decltype(IState::x[0] + 0);
    const Elem (*gs)[32] = reinterpret_cast<const Elem (*)[32]>(gs_raw);
    const int lane = threadIdx.x & 31;
    IState S;
#pragma unroll
    for (int k = 0; k < R_I; ++k) { S.x[k] = gs[k][lane]; S.y[k] = gs[R_I + k][lane]; S.z[k] = gs[2 * R_I + k][lane]; S.h[k] = gs[3 * R_I + k][lane]; }
    if constexpr (BOX == 2) Path::near_images(*T, S, acc, L, invL, img_tab, j0, j1);
    else Path::template near_global<BOX == 1>(*T, S, acc, L, invL, j0, j1);
}

template <typename Path, int BOX>
__global__ void __launch_bounds__(CTA_THREADS, 1)
forces_boxring_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                      const typename Path::Tile* __restrict__ tiles, int nt, double* __restrict__ acc_out,
                      double* __restrict__ partials, int zero, double box_L, double box_invL,
                      const GroupMeta* __restrict__ gm, const SymPlan* __restrict__ plan, double* __restrict__ acc_lo_out)
{
    const bool restricted = plan != nullptr && plan->W < plan->nb - 1;
    const int my_block = (int)(((long long)blockIdx.x * SPLITJ_GROUP) / IB);
    using Tile = typename Path::Tile;
    using IState = typename Path::IState;
    using Elem = decltype(IState::x[0] + 0);               // double or float
    static_assert(BOX == 1 || (BOX == 2 && Path::NOUT == 6), "leading image (both paths) or image sum (fp64)");
    constexpr int G = BOXRING_G, STAGES = boxring_stages<Path, BOX>(), FAR_BYTES = boxring_part_bytes<Path, BOX>();
    constexpr size_t PART_OFFSET = BOX == 2 ? TJ * sizeof(FarSrcF64) : 0;      // of the carried part within the tile record
    constexpr int WARPS = CTA_THREADS / 32, WG = WARPS / G, PER_WARP = TJ / WG;   // 4 warps per sub-ring, 64 sources per warp and tile
    static_assert(WARPS % G == 0 && TJ % WG == 0 && PER_WARP % 4 == 0, "every warp takes whole float4 groups of each tile");
    static_assert(FAR_BYTES % 128 == 0 && PART_OFFSET % 16 == 0, "stage alignment");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[G][STAGES], empty_bar[G][STAGES];
    __shared__ Elem gs[4 * R_I][32];                        // the group's particles (x, y, z, h), unshifted: read back when a
                                                            // tile needs another image shift or the general body
    // BOX = 2: image offsets n L of the unpruned route (near_images), of all n in [-3, 3]^3 (pruned route), and per warp the
    // candidates of its current tile
    constexpr int NCUBE = 343, CAND_STRIDE = 352;
    __shared__ double img_tab[BOX == 2 ? 3 * EWALD_NTRIPLETS : 1];
    __shared__ double cube_tab[BOX == 2 ? 3 * NCUBE : 1];
    __shared__ unsigned short cand_all[BOX == 2 ? WARPS * CAND_STRIDE : 1];
    if constexpr (BOX == 2) {
        for (int q = threadIdx.x; q < EWALD_NTRIPLETS; q += CTA_THREADS) {
            img_tab[3 * q] = ewald_triplets[q].x * box_L; img_tab[3 * q + 1] = ewald_triplets[q].y * box_L;
            img_tab[3 * q + 2] = ewald_triplets[q].z * box_L;
        }
        for (int q = threadIdx.x; q < NCUBE; q += CTA_THREADS) {
            cube_tab[3 * q] = (double)(q % 7 - 3) * box_L; cube_tab[3 * q + 1] = (double)((q / 7) % 7 - 3) * box_L;
            cube_tab[3 * q + 2] = (double)(q / 49 - 3) * box_L;
        }
    }
    double* acc_all = reinterpret_cast<double*>(smem_raw + G * STAGES * FAR_BYTES);   // [NOUT * R_I][CTA_THREADS]
    double* acc = acc_all + threadIdx.x;
    uint32_t* codes_all = reinterpret_cast<uint32_t*>(acc_all + Path::NOUT * R_I * CTA_THREADS);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = warp / WG, wg = warp % WG;                 // sub-ring, warp within it
    unsigned char* ring = smem_raw + g * STAGES * FAR_BYTES;
    const uint32_t* codes = codes_all + g * DEC_CHUNK;
    const bool producer = wg == 0 && lane == 0;

    // the group's bounds (bounding box, largest softening) live in shared memory, not in registers: they
    // are needed once per chunk (and per tile in the image sum), and the far loops need every register
    __shared__ float gbox[8];                               // lo[3], hi[3], hmax
    {
        IState S;
        float blo[3], bhi[3], hh, rlo, rhi;
        const long long i0 = (long long)blockIdx.x * SPLITJ_GROUP + lane;     // the same particles in every warp
        load_i_block<Path>(S, pos, soft, N, i0, N, rlo, rhi, hh);
        warp_box<Path>(S, blo, bhi);
        if (warp == 0) {
#pragma unroll
            for (int k = 0; k < R_I; ++k) { gs[k][lane] = S.x[k]; gs[R_I + k][lane] = S.y[k]; gs[2 * R_I + k][lane] = S.z[k]; gs[3 * R_I + k][lane] = S.h[k]; }
            if (lane == 0) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { gbox[c] = blo[c]; gbox[3 + c] = bhi[c]; }
                gbox[6] = hh;
            }
        }
    }
    auto group_state = [&]() {
        IState S;
#pragma unroll
        for (int k = 0; k < R_I; ++k) { S.x[k] = gs[k][lane]; S.y[k] = gs[R_I + k][lane]; S.z[k] = gs[2 * R_I + k][lane]; S.h[k] = gs[3 * R_I + k][lane]; }
        return S;
    };
#pragma unroll
    for (int q = 0; q < Path::NOUT * R_I; ++q) acc[q * CTA_THREADS] = 0.0;

    // The tiles of this CTA: first, first + step, ... (`ntiles` of them) -- every gridDim.y-th tile, so that the CTAs that
    // share a group meet the same mix of decisions; restricted mode: the tiles of the group's own block (gridDim.y = 1).
    // Sub-ring g takes every G-th of those, for the same reason: the four finish together.
    const int first = restricted ? min(nt, my_block * (IB / TJ)) : (int)blockIdx.y;
    const int step = restricted ? 1 : (int)gridDim.y;
    const int ntiles = restricted ? min(nt, (my_block + 1) * (IB / TJ)) - first : (nt - first + step - 1) / step;
    auto tile_of = [&](int r, int k) { return first + step * (r + G * k); };      // tile k of sub-ring r
    const int mine = (ntiles - g + G - 1) / G;               // tiles of this sub-ring
    const int chunks = ((ntiles + G - 1) / G + DEC_CHUNK - 1) / DEC_CHUNK;    // the same for every sub-ring (CTA-wide barriers)
    if (threadIdx.x == 0) {
#pragma unroll
        for (int r = 0; r < G; ++r)
#pragma unroll
            for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[r][s], 1); mbar_init(&empty_bar[r][s], WG); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    typename Path::FarSums F;
    init_far_sums<Path>(F, acc);
    Path::far_zero(F);
    IState Q;                                               // the group with the current image shift on it
    uint32_t q_key = 0xffffffffu;                           // the shift bytes Q was built for (none yet)
    int pending = 0;                                        // sources summed in F since its last flush
    int produced = 0, consumed = 0;                         // far tiles of this sub-ring so far
    const int j0 = wg * PER_WARP, j1 = j0 + PER_WARP;
    for (int ch = 0; ch < chunks; ++ch) {
        const int k0 = ch * DEC_CHUNK, cnt = max(0, min(DEC_CHUNK, mine - k0));   // this sub-ring's tiles k0 .. k0 + cnt of its list
        __syncthreads();                                    // the previous chunk's decisions are no longer read (and: gs, barrier init)
        const float blo[3] = {gbox[0], gbox[1], gbox[2]}, bhi[3] = {gbox[3], gbox[4], gbox[5]};
        const float hh = gbox[6];
        for (int q = threadIdx.x; q < G * DEC_CHUNK; q += CTA_THREADS) {       // all threads compute the decisions of all sub-rings
            const int r = q / DEC_CHUNK, k = k0 + q % DEC_CHUNK;
            if (r + G * k < ntiles)
                codes_all[q] = boxcode_pack(box_shift(blo, bhi, hh, tiles[tile_of(r, k)].meta, box_L, box_invL), box_invL);
        }
        __syncthreads();
        int pq = 0;                                         // producer cursor within the chunk
        auto produce_next = [&]() {                         // the next far tile of the chunk, if any
            while (pq < cnt && (codes[pq] & BOXCODE_GENERAL)) ++pq;
            if (pq >= cnt) return;
            const int s = produced % STAGES;
            if (produced >= STAGES) mbar_wait(&empty_bar[g][s], ((produced / STAGES) - 1) & 1);
            mbar_expect_tx(&full_bar[g][s], (uint32_t)FAR_BYTES);
            bulk_load(ring + s * FAR_BYTES, reinterpret_cast<const unsigned char*>(tiles + tile_of(g, k0 + pq)) + PART_OFFSET,
                      (uint32_t)FAR_BYTES, &full_bar[g][s]);
            ++produced; ++pq;
        };
        if (producer)
            for (int k = 0; k < STAGES - 1; ++k) produce_next();
        for (int q = 0; q < cnt; ++q) {
            const uint32_t code = codes[q];
            if (code & BOXCODE_GENERAL) {
                if constexpr (BOX != 2) { if (pending) { Path::fold_flush(F, acc); pending = 0; } }
                boxring_general<Path, BOX>(&tiles[tile_of(g, k0 + q)], &gs[0][0], acc, box_L, box_invL, img_tab, j0, j1);
                continue;
            }
            if (producer) produce_next();
            const int s = consumed % STAGES;
            mbar_wait(&full_bar[g][s], (consumed / STAGES) & 1);
            if constexpr (BOX == 2) {
                // the candidate images of this warp's 64 sources of the tile against the group, pruned from the two bounding
                // boxes (see the header comment); the sources' box is taken from the staged copy itself -- a quarter of a
                // cell-ordered tile is more compact than the tile, and every candidate less is 1 % of the work
                const double* P = reinterpret_cast<const double*>(ring + s * FAR_BYTES);      // x[], y[], z[], m[], h[]
                double sh[3], a[3], b[3];
                const double eps = 1.0e-5 * box_L;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double lo = __longlong_as_double(0x7ff0000000000000ll), hi = -lo;
#pragma unroll
                    for (int r = 0; r < PER_WARP / 32; ++r) {
                        const int j = j0 + 32 * r + lane;
                        if (P[3 * TJ + j] != 0.0) { lo = fmin(lo, P[c * TJ + j]); hi = fmax(hi, P[c * TJ + j]); }    // pads (m = 0) are parked
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) { lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
                    const double dmin = (lo - (double)gbox[3 + c]) - eps, dmax = (hi - (double)gbox[c]) + eps;
                    sh[c] = box_L * rint(0.5 * (dmin + dmax) * box_invL);
                    a[c] = dmin - sh[c]; b[c] = dmax - sh[c];
                }
                unsigned short* cand = cand_all + warp * CAND_STRIDE;
                const double cut2 = (2.6 * box_L) * (2.6 * box_L);
                int ncand = 0;
                for (int q0 = 0; q0 < NCUBE; q0 += 32) {
                    const int t = q0 + lane;
                    bool keep = false;
                    if (t < NCUBE) {
                        double g2 = 0.0;
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            const double o = cube_tab[3 * t + c];
                            const double gap = fmax(0.0, fmax(a[c] - o, o - b[c]));
                            g2 = fma(gap, gap, g2);
                        }
                        keep = g2 < cut2;
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, keep);
                    if (keep) cand[ncand + __popc(m & ((1u << lane) - 1u))] = (unsigned short)t;
                    ncand += __popc(m);
                }
                __syncwarp();
                Q = group_state();
#pragma unroll
                for (int k = 0; k < R_I; ++k) { Q.x[k] += sh[0]; Q.y[k] += sh[1]; Q.z[k] += sh[2]; }
                Path::far_images(P, P + TJ, P + 2 * TJ, P + 3 * TJ, Q, acc, box_L, cube_tab, cand, ncand, j0, j1);
            } else {
                const Tile& T = *reinterpret_cast<const Tile*>(ring + s * FAR_BYTES);    // only its far part is there
                if ((code >> 8) != q_key) {
                    q_key = code >> 8;
                    Q = Path::shifted(group_state(), boxcode_unpack(code, box_L).s);
                }
                far_fold_dispatch<Path>(T, Q, F, zero, (int)(code & 7u), 0.5 * box_L, j0, j1);
                pending += PER_WARP;
                if (pending >= Path::FAR_SOURCES_PER_FLUSH) { Path::fold_flush(F, acc); pending = 0; }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[g][s]);
            ++consumed;
        }
    }
    if (pending) Path::fold_flush(F, acc);
    __syncthreads();

    // fixed-order sum over the 16 warps: thread (c, k, l) owns component c of particle l + 32 k of the group
    if (threadIdx.x < 3 * SPLITJ_GROUP) {
        const int c = threadIdx.x / SPLITJ_GROUP, r = threadIdx.x % SPLITJ_GROUP, k = r / 32, l = r % 32;
        double hi = 0.0, lo = 0.0;
        for (int w = 0; w < WARPS; ++w) {
            const double v = acc_all[(c * R_I + k) * CTA_THREADS + w * 32 + l];
            const double s = hi + v, bb = s - hi;
            lo += (hi - (s - bb)) + (v - bb);                              // TwoSum
            hi = s;
            if (Path::NOUT == 6) lo += acc_all[((3 + c) * R_I + k) * CTA_THREADS + w * 32 + l];
        }
        const long long i = (long long)blockIdx.x * SPLITJ_GROUP + l + 32 * k;
        if (gridDim.y == 1) {
            if (i < N) {
                if (acc_lo_out) {
                    if (restricted) {                                        // += what forces_boxgen_kernel left there
                        const double v = acc_out[(long long)c * N + i];
                        const double s = hi + v, bb = s - hi;
                        lo += (hi - (s - bb)) + (v - bb) + acc_lo_out[(long long)c * N + i];
                        hi = s;
                    }
                    acc_out[(long long)c * N + i] = hi; acc_lo_out[(long long)c * N + i] = lo;
                } else acc_out[(long long)c * N + i] = hi + lo;
            }
        } else {
            double* rec = partials + (((long long)blockIdx.x * gridDim.y + blockIdx.y) * 6) * SPLITJ_GROUP;
            rec[c * SPLITJ_GROUP + r] = hi; rec[(3 + c) * SPLITJ_GROUP + r] = lo;
        }
    }
}

// ---- the possibly-softened units of other blocks (periodic pair-symmetric evaluation) -----------------------------------
// One 128-particle group per CTA.  pair_decision (common.cuh) is taken for the group (fp64) / its 256-particle parent
// (mixed) against every 128- / 256-source unit of the OTHER blocks -- the very call by which forces_sym_box_kernel skips
// a meeting; the units it calls "general" are gathered into a list in a fixed order (warp w scans its slice of the units,
// the offsets come from the warps' counts); the listed units' plain sources are staged in shared memory eight at a time
// and each is shared by four warps (a quarter of its sources each) through the general wrapped body.  Writes the group's
// result double-double (zero when the plan has no items: then forces_boxring_kernel evaluates everything).
// gridDim.y > 1 splits the unit range over CTAs (records [group][y][6][128] in `records`, summed by forces_splitj_reduce):
// a group whose bounding box spans the whole box -- its 128 particles straddle a top-level jump of the cell order, a few
// groups of any set -- has EVERY unit on its list, and one CTA would work on it long after all others are done.
constexpr int BOXGEN_CHUNK = 4096;                         // units decided and listed at a time (16 KiB of list)
constexpr int BOXGEN_BATCH = 8;                            // listed units staged in shared memory at a time (5 KiB each)
template <typename Path>
constexpr int boxgen_smem_bytes()
{
    return Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double) + BOXGEN_CHUNK * (int)sizeof(uint32_t) +
           BOXGEN_BATCH * 5 * (Path::NOUT == 6 ? 1 : 2) * SPLITJ_GROUP * (Path::NOUT == 6 ? 8 : 4);
}

// BOX = 2: the same for the image sum (the listed units through Fp64Path::near_images_view, all 179 candidates).
template <typename Path, int BOX = 1>
__global__ void __launch_bounds__(CTA_THREADS, 1)
forces_boxgen_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                     const typename Path::Tile* __restrict__ tiles, int nt, double* __restrict__ acc_hi, double* __restrict__ acc_lo,
                     double* __restrict__ records, double box_L, double box_invL, const GroupMeta* __restrict__ gm,
                     const SymPlan* __restrict__ plan)
{
    using IState = typename Path::IState;
    __shared__ double img_tab[BOX == 2 ? 3 * EWALD_NTRIPLETS : 1];
    if constexpr (BOX == 2) {
        for (int q = threadIdx.x; q < EWALD_NTRIPLETS; q += CTA_THREADS) {
            img_tab[3 * q] = ewald_triplets[q].x * box_L; img_tab[3 * q + 1] = ewald_triplets[q].y * box_L;
            img_tab[3 * q + 2] = ewald_triplets[q].z * box_L;
        }
    }
    constexpr int GRAN = Path::NOUT == 6 ? 1 : 2;           // groups per unit (the symmetric kernels' subgroups)
    using Elem = decltype(IState::x[0] + 0);                // double or float
    constexpr int UNIT = GRAN * SPLITJ_GROUP, WARPS = CTA_THREADS / 32, WPU = 4, SLICE = UNIT / WPU;   // 4 warps per unit
    static_assert(TJ == 2 * SPLITJ_GROUP && SLICE % 2 == 0, "a tile is two groups; the mixed general body takes sources in pairs");
    static_assert(BOXGEN_BATCH % (WARPS / WPU) == 0, "whole rounds of WARPS / WPU units per batch");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ int gcount[(BOXGEN_CHUNK / CTA_THREADS) * WARPS];
    double* acc_all = reinterpret_cast<double*>(smem_raw);
    double* acc = acc_all + threadIdx.x;
    uint32_t* glist = reinterpret_cast<uint32_t*>(acc_all + Path::NOUT * R_I * CTA_THREADS);
    Elem* stage = reinterpret_cast<Elem*>(glist + BOXGEN_CHUNK);             // [BOXGEN_BATCH][5 (x, y, z, m, h)][UNIT]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool active = plan->W < plan->nb - 1;
    const int my_block = (int)(((long long)blockIdx.x * SPLITJ_GROUP) / IB);
    const int me = (int)blockIdx.x / GRAN;                  // this group's unit index
    const int units_all = (int)((N + UNIT - 1) / UNIT);
    const int u_lo = (int)((long long)blockIdx.y * units_all / gridDim.y), units = (int)(((long long)blockIdx.y + 1) * units_all / gridDim.y);

    IState S;
    {
        float rlo, rhi, hh;
        const long long i0 = (long long)blockIdx.x * SPLITJ_GROUP + lane;
        load_i_block<Path>(S, pos, soft, N, i0, N, rlo, rhi, hh);
    }
#pragma unroll
    for (int q = 0; q < Path::NOUT * R_I; ++q) acc[q * CTA_THREADS] = 0.0;

    for (int u0 = u_lo; active && u0 < units; u0 += BOXGEN_CHUNK) {
        const int cnt = min(BOXGEN_CHUNK, units - u0);
        constexpr int ROUNDS = BOXGEN_CHUNK / CTA_THREADS;  // decisions per thread: unit q = r * CTA_THREADS + thread
        auto wanted = [&](int q) {
            if (q >= cnt) return false;
            const int u = u0 + q;
            if constexpr (BOX == 2) {
                // the image-sum kernel softens in place and takes the groups' own blocks as well (diagonal items): left are the
                // group's meeting with itself and the meetings whose boxes span a period
                return u == me || pair_too_wide<GRAN>(gm, me, u, box_L);
            } else {
                if ((int)(((long long)u * UNIT) / IB) == my_block) return false;   // own block: forces_boxring_kernel
                return (boxcode_pack(pair_decision<GRAN>(gm, me, u, box_L, box_invL), box_invL) & BOXCODE_GENERAL) != 0;
            }
        };
        // (thread-interleaved: a CTA's share of a group is usually a few hundred units, one decision per thread; the list
        // is in unit order: the offsets come from the (round, warp) counts)
        unsigned flags[ROUNDS];
        __syncthreads();                                    // the previous chunk's list and counts are no longer read
#pragma unroll
        for (int r = 0; r < ROUNDS; ++r) {
            flags[r] = r * CTA_THREADS < cnt ? __ballot_sync(0xffffffffu, wanted(r * CTA_THREADS + threadIdx.x)) : 0u;
            if (lane == 0) gcount[r * WARPS + warp] = __popc(flags[r]);
        }
        __syncthreads();
        int total_cnt = 0;
        {
            int at = 0;
#pragma unroll
            for (int r = 0; r < ROUNDS; ++r) {
                int before = 0;
                for (int w = 0; w < WARPS; ++w) { const int c = gcount[r * WARPS + w]; if (w < warp) before += c; total_cnt += c; }
                if (flags[r] >> lane & 1u) glist[at + before + __popc(flags[r] & ((1u << lane) - 1u))] = (uint32_t)(u0 + r * CTA_THREADS + threadIdx.x);
                for (int w = 0; w < WARPS; ++w) at += gcount[r * WARPS + w];
            }
        }
        __syncthreads();
        for (int e0 = 0; e0 < total_cnt; e0 += BOXGEN_BATCH) {
            const int nbatch = min(BOXGEN_BATCH, total_cnt - e0);
            if (e0 > 0) __syncthreads();                    // the previous batch is no longer read
            for (int q = threadIdx.x; q < nbatch * 5 * UNIT; q += CTA_THREADS) {
                const int e = q / (5 * UNIT), a = (q / UNIT) % 5, j = q % UNIT;
                const long long src = (long long)glist[e0 + e] * UNIT;            // first source of the unit
                // x[], y[], z[], m[], h[] follow one another in the tile record (common.cuh)
                stage[q] = (&tiles[src / TJ].x[0])[a * TJ + (int)(src % TJ) + j];
            }
            __syncthreads();
            for (int e = warp / WPU; e < nbatch; e += WARPS / WPU) {
                const Elem* u = stage + e * 5 * UNIT;
                const int j0 = (warp % WPU) * SLICE;
                if constexpr (BOX == 2)
                    Path::near_images_view(u, u + UNIT, u + 2 * UNIT, u + 3 * UNIT, u + 4 * UNIT, S, acc, box_L, box_invL, img_tab, j0, j0 + SLICE);
                else
                    Path::template near_view<true>(u, u + UNIT, u + 2 * UNIT, u + 3 * UNIT, u + 4 * UNIT, S, acc, box_L, box_invL, j0, j0 + SLICE);
            }
        }
    }
    __syncthreads();
    if (threadIdx.x < 3 * SPLITJ_GROUP) {                   // fixed-order sum over the 16 warps, as in the split-j driver
        const int c = threadIdx.x / SPLITJ_GROUP, r = threadIdx.x % SPLITJ_GROUP, k = r / 32, l = r % 32;
        double hi = 0.0, lo = 0.0;
        for (int w = 0; w < WARPS; ++w) {
            const double v = acc_all[(c * R_I + k) * CTA_THREADS + w * 32 + l];
            const double s = hi + v, bb = s - hi;
            lo += (hi - (s - bb)) + (v - bb);                              // TwoSum
            hi = s;
            if (Path::NOUT == 6) lo += acc_all[((3 + c) * R_I + k) * CTA_THREADS + w * 32 + l];
        }
        const long long i = (long long)blockIdx.x * SPLITJ_GROUP + l + 32 * k;
        if (gridDim.y == 1) {
            if (i < N) { acc_hi[(long long)c * N + i] = hi; acc_lo[(long long)c * N + i] = lo; }
        } else {
            double* rec = records + (((long long)blockIdx.x * gridDim.y + blockIdx.y) * 6) * SPLITJ_GROUP;
            rec[c * SPLITJ_GROUP + r] = hi; rec[(3 + c) * SPLITJ_GROUP + r] = lo;
        }
    }
}

// ---- simple driver (cross-check) -----------------------------------------------------------------
template <typename Path>
__global__ void __launch_bounds__(CTA_THREADS, 1)
forces_v1_kernel(const double* __restrict__ pos, const double* __restrict__ soft, long long N,
                 const typename Path::Tile* __restrict__ tiles, int ntiles, long long i_begin, long long i_end,
                 double* __restrict__ acc_out, int zero)
{
    using Tile = typename Path::Tile;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Tile& tile = *reinterpret_cast<Tile*>(smem_raw);
    double* acc = reinterpret_cast<double*>(smem_raw + stage_stride((int)sizeof(Tile))) + threadIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long i0 = i_begin + (long long)blockIdx.x * IB + (long long)warp * WARP_I + lane;
    typename Path::IState S;
    float rlo, rhi, hh;
    load_i_block<Path>(S, pos, soft, N, i0, i_end, rlo, rhi, hh);
#pragma unroll
    for (int q = 0; q < Path::NOUT * R_I; ++q) acc[q * CTA_THREADS] = 0.0;
    for (int t = 0; t < ntiles; ++t) {
        __syncthreads();
        {
            const uint4* src = reinterpret_cast<const uint4*>(tiles + t);
            uint4* dst = reinterpret_cast<uint4*>(&tile);
            for (int q = threadIdx.x; q < (int)(sizeof(Tile) / 16); q += CTA_THREADS) dst[q] = src[q];
        }
        __syncthreads();
        if (tile_is_far(rlo, rhi, hh, tile.meta)) {
            typename Path::FarSums F;
            init_far_sums<Path>(F, acc);
            Path::far(tile, S, F, zero);
            Path::far_flush(F, acc);                       // the cross-check driver flushes at every tile
        } else {
            Path::near(tile, S, acc);
        }
    }
    const long long cnt = i_end - i_begin;
#pragma unroll
    for (int k = 0; k < R_I; ++k) {
        const long long i = i0 + 32 * k;
        if (i < i_end) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double v = acc[(c * R_I + k) * CTA_THREADS];
                if (Path::NOUT == 6) v += acc[((3 + c) * R_I + k) * CTA_THREADS];
                acc_out[(long long)c * cnt + (i - i_begin)] = v;
            }
        }
    }
}

}  // namespace steps
