// steps.cu -- C ABI of steps-b200 (include/steps.h): argument checks, workspace, launches.
// Every step of the hot path runs in the kernels of this translation unit; there is no CPU
// fallback and no dependency on oracle/.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/steps.h"
#include "common.cuh"
#include "prep.cuh"
#include "force_mixed.cuh"
#include "force_fp64.cuh"
#include "force_driver.cuh"
#include "force_sym.cuh"
#include "kdk.cuh"
#include "sort.cuh"

using namespace steps;

namespace {

std::atomic<long long> g_launches{0};
// Eq. 12 fused into the last kernel of the force evaluation that steps_kdk_step_adaptive launches (Eq12Fuse, common.cuh):
// set by that call around its forces_impl, read by the launchers of the final-writer kernels of FULL evaluations.
thread_local Eq12Fuse t_fuse = {nullptr, nullptr, nullptr, 0.0, 0.0, 0.0, nullptr};
const Eq12Fuse NO_FUSE = {nullptr, nullptr, nullptr, 0.0, 0.0, 0.0, nullptr};
thread_local int g_last_cuda_error = 0;
std::atomic<int> g_driver{0};   // 0 = default, 1 = simple v1 driver (cross-check)
std::atomic<int> g_profile{0};  // 1 = bracket the force kernel with CUDA events on its stream

constexpr int MAX_DEVICES = 16;
#ifndef STEPS_STAGES
#define STEPS_STAGES 4
#endif
constexpr int STAGES = STEPS_STAGES;   // depth of the bulk-copy ring
constexpr int MAX_GRID = 148 * 4;

// Pair-symmetric evaluation (force_sym.cuh) of the fp64 path: used for full evaluations of at least SYM_MIN_BLOCKS blocks;
// its partial records are produced and consumed in panels of at most g_sym_panel_items items (96 KiB of records each).
constexpr int SYM_MIN_BLOCKS = 9;          // fp64: from N = 16,385, with the items split into parts while the blocks are few
constexpr int SYM_BOX_MIN_BLOCKS = 9;      // periodic boxes, fp64 (leading image and image sum): from N = 16,385 as well
constexpr int SYM_SPLITJ_BAND_MAX_BLOCKS = 64;   // up to here the band of a pair-symmetric evaluation runs on the split-j driver
constexpr int SYM_MIN_BLOCKS_MIXED = 16;   // mixed: from N = 30,721 too; whole items from 24 blocks (N >= 47,105), below that each item in 4 parts
constexpr int SYM_BOX_MIN_BLOCKS_MIXED = 80;       // periodic boxes, mixed: N >= 161,793 (measured crossover with the group-ring kernel)
constexpr int SYM_MIXED_WHOLE_ITEMS_BLOCKS = 24;   // (the split variant of the mixed kernel is slower per pair: measured, profiles/r02_sizes.md)
std::atomic<long long> g_sym_panel_items{16384};
std::atomic<int> g_sym_enabled{1};
std::atomic<int> g_splitj{1};           // 0 = never use the split-j driver (testing)
std::atomic<int> g_box_gsplit{8};       // CTAs per group in forces_boxgen_kernel (option "box_gsplit", tuning)

// What the fused Eq. 12 minimum of the last steps_kdk_step_adaptive call was computed from (see that function).
struct FuseToken {
    const void *pos, *acc, *soft, *state;
    long long N;
    double absG, B, eps;
    long long launches;
    bool operator==(const FuseToken& o) const
    {
        return pos == o.pos && acc == o.acc && soft == o.soft && state == o.state && N == o.N && absG == o.absG && B == o.B &&
               eps == o.eps && launches == o.launches;
    }
};
std::atomic<int> g_fuse_eq12{1};        // 0 = always the separate Eq. 12 pass (testing)

struct Workspace {
    void* tiles = nullptr;          // max(sizeof(TileF32), sizeof(TileF64)) * ntiles (padded to whole blocks)
    double* partials = nullptr;     // (nb + grid) * 6 * IB doubles (persistent driver's split-j records)
    long long cap_particles = 0;
    SymPlan* plan = nullptr;        // SymPlan + its arrays (sym_plan_bytes)
    GroupMeta* gm = nullptr;        // one per 128 particles, padded to whole blocks (periodic pair-symmetric evaluation)
    double* acc_dd = nullptr;       // 6 N doubles: (hi, lo) of the band result, the symmetric records are added to it
    double* sym_records = nullptr;  // 2 * panel_items * 3 * IB doubles (row records, then column records)
    long long sym_cap_particles = 0, sym_panel_items = 0;
    int num_sms = 0;
    int grid_mixed = 0, grid_fp64 = 0, grid_fp64_band = 0, grid_mixed_band = 0, grid_sym = 0, grid_sym_mixed = 0;   // persistent grids: SMs x resident CTAs
    double* mom_partial = nullptr;  // MOM_BLOCKS * 4
    void* sort_buf = nullptr;       // steps_sort_radial: keys in/out, index in, cub temporary storage
    size_t sort_bytes = 0;
    // staging buffers of steps_forces_host
    double* h_pos = nullptr; double* h_mass = nullptr; double* h_soft = nullptr; double* h_acc = nullptr;
    long long h_cap = 0;
    int cc_major = -1;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;   // "profile" option: around the last force kernel(s)
    bool ev_valid = false;
    bool sym_split_ready = false, sym_split_ready_mixed = false;
    FuseToken fuse_token{};
    bool fuse_valid = false;
    // One scratch area per device: calls on different streams are serialised through this event (see claim_scratch).
    cudaEvent_t scratch_done = nullptr;
    cudaStream_t scratch_stream = nullptr;
    bool scratch_used = false;
};
Workspace g_ws[MAX_DEVICES];
std::mutex g_mutex;

inline long long nblocks_of(long long cnt) { return (cnt + IB - 1) / IB; }
inline long long ntiles_of(long long N) { return (N + TJ - 1) / TJ; }
inline long long ntiles_padded(long long N) { return nblocks_of(N) * TPB; }       // whole blocks (force_sym.cuh)
inline size_t partial_bytes(long long N) { return sizeof(double) * 6 * IB * (size_t)(nblocks_of(N) + MAX_GRID); }
inline size_t tile_bytes_max() { return sizeof(TileF64) > sizeof(TileF32) ? sizeof(TileF64) : sizeof(TileF32); }
inline long long sym_items_max(long long N) { const long long nb = nblocks_of(N); return nb * (nb - 1) / 2; }
inline long long sym_panel_items_for(long long N) { return std::max(1ll, std::min(16 * sym_items_max(N), g_sym_panel_items.load())); }
inline size_t sym_record_bytes(long long items) { return sizeof(double) * 2 * 3 * IB * (size_t)items; }
inline bool sym_eligible(long long N, bool mixed = false)
{
    return g_sym_enabled.load() != 0 && nblocks_of(N) >= (mixed ? SYM_MIN_BLOCKS_MIXED : SYM_MIN_BLOCKS);
}

int cuda_fail(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    return STEPS_ECUDA;
}
#define STEPS_CUDA(call)                                   \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return cuda_fail(e__);     \
    } while (0)

int current_device(int* dev)
{
    STEPS_CUDA(cudaGetDevice(dev));
    if (*dev < 0 || *dev >= MAX_DEVICES) return STEPS_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mutex);
    Workspace& w = g_ws[*dev];
    if (w.cc_major < 0) {
        int major = 0;
        STEPS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, *dev));
        STEPS_CUDA(cudaDeviceGetAttribute(&w.num_sms, cudaDevAttrMultiProcessorCount, *dev));
        w.cc_major = major;
    }
    if (w.cc_major != 10) return STEPS_EUNSUPPORTED;   // sm_100a cubin only
    return STEPS_OK;
}

bool stream_is_capturing(cudaStream_t st)
{
    cudaStreamCaptureStatus status = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &status) != cudaSuccess) { cudaGetLastError(); return false; }
    return status != cudaStreamCaptureStatusNone;
}

// (Re)allocates the per-device scratch for N particles.  Never allocates while `st` is being captured into a CUDA graph
// (cudaMalloc/cudaFree are not capturable): STEPS_ECAPTURE tells the caller to steps_reserve(N) before the capture.
int ensure_workspace(int dev, long long N, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    Workspace& w = g_ws[dev];
    const bool need_small = !w.mom_partial;
    const bool need_tiles = N > w.cap_particles;
    const bool need_sym = sym_eligible(N) && (N > w.sym_cap_particles || sym_panel_items_for(N) > w.sym_panel_items);
    if (!need_small && !need_tiles && !need_sym) return STEPS_OK;
    if (stream_is_capturing(st)) return STEPS_ECAPTURE;
    if (need_small) {
        // first use of this device: the reduction scratch and the image-sum triplet table (Eq. 5) in constant memory
        static const EwaldTriplets table;
        STEPS_CUDA(cudaMemcpyToSymbol(ewald_triplets, table.v, sizeof(table.v)));
        if (cudaMalloc(&w.mom_partial, sizeof(double) * MOM_BLOCKS * 4) != cudaSuccess) { cudaGetLastError(); return STEPS_ENOMEM; }
    }
    if (need_tiles || need_sym) STEPS_CUDA(cudaDeviceSynchronize());      // nothing in flight may still use the old scratch
    if (need_tiles) {
        cudaFree(w.tiles); cudaFree(w.partials); cudaFree(w.plan); cudaFree(w.gm);
        w.tiles = nullptr; w.partials = nullptr; w.plan = nullptr; w.gm = nullptr; w.cap_particles = 0;
        if (cudaMalloc(&w.tiles, tile_bytes_max() * (size_t)ntiles_padded(N)) != cudaSuccess ||
            cudaMalloc(&w.partials, partial_bytes(N)) != cudaSuccess ||
            cudaMalloc(&w.plan, sym_plan_bytes(nblocks_of(N))) != cudaSuccess ||
            cudaMalloc(&w.gm, sizeof(GroupMeta) * (size_t)nblocks_of(N) * (IB / SPLITJ_GROUP)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(w.tiles); cudaFree(w.partials); cudaFree(w.plan); w.tiles = nullptr; w.partials = nullptr; w.plan = nullptr;
            return STEPS_ENOMEM;
        }
        w.cap_particles = nblocks_of(N) * IB;
    }
    if (need_sym) {
        cudaFree(w.acc_dd); cudaFree(w.sym_records);
        w.acc_dd = nullptr; w.sym_records = nullptr; w.sym_cap_particles = 0; w.sym_panel_items = 0;
        const long long items = sym_panel_items_for(N);
        if (cudaMalloc(&w.acc_dd, sizeof(double) * 6 * (size_t)N) != cudaSuccess ||
            cudaMalloc(&w.sym_records, sym_record_bytes(items)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(w.acc_dd); w.acc_dd = nullptr;
            return STEPS_ENOMEM;
        }
        w.sym_cap_particles = N; w.sym_panel_items = items;
    }
    return STEPS_OK;
}

// The scratch area (tiles, partial records, reduction partials, run coefficients) is ONE per device.  Calls are
// stream-ordered on their own stream; a call on a DIFFERENT stream than the previous user first waits (on the device,
// cudaStreamWaitEvent) for the previous user's last kernel, so concurrent streams are serialised instead of racing.
// Streams under graph capture are left alone (events cannot cross a capture): one capturing stream per device at a time.
int claim_scratch(Workspace& w, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (stream_is_capturing(st)) return STEPS_OK;
    if (!w.scratch_done) STEPS_CUDA(cudaEventCreateWithFlags(&w.scratch_done, cudaEventDisableTiming));
    if (w.scratch_used && w.scratch_stream != st) STEPS_CUDA(cudaStreamWaitEvent(st, w.scratch_done, 0));
    return STEPS_OK;
}
int release_scratch(Workspace& w, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (stream_is_capturing(st)) return STEPS_OK;
    STEPS_CUDA(cudaEventRecord(w.scratch_done, st));
    w.scratch_stream = st; w.scratch_used = true;
    return STEPS_OK;
}

bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

template <typename Kernel>
int persistent_grid(Kernel kern, int smem, const Workspace& w, int& grid_cache, int threads = CTA_THREADS)
{
    if (grid_cache == 0) {
        STEPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        int per_sm = 0;
        STEPS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem));
        if (per_sm < 1) return STEPS_EUNSUPPORTED;
        const int g = w.num_sms * per_sm;
        grid_cache = g > MAX_GRID ? MAX_GRID : g;
    }
    return STEPS_OK;
}

// Full evaluation, pair-symmetric (force_sym.cuh): band through the asymmetric persistent kernel, every far block pair once
// through the symmetric kernel, panel by panel; all decisions that depend on the data (W) are taken on the device.
template <typename Path>
int launch_forces_sym(const double* pos, const double* mass, const double* soft, long long N, double* acc_out,
                      cudaStream_t st, Workspace& w, int share_rank = 0, int share_world = 1)
{
    // share_world > 1 (steps_forces_share): the share_rank-th of share_world equal parts of the WORK -- of the band's tile
    // visits and of the symmetric (sub-)items, both counted on the device -- with acc_out = this part's contribution to
    // every particle's acceleration.
    using Tile = typename Path::Tile;
    constexpr bool FP64 = Path::NOUT == 6;
    const int nb = (int)nblocks_of(N);
    const int ntp = nb * TPB;
    Tile* tiles = reinterpret_cast<Tile*>(w.tiles);
    constexpr int smem_band = persistent_smem_bytes<Path, STAGES>();
    auto band = forces_persistent_kernel<Path, STAGES, 0, true>;
    int rc = persistent_grid(band, smem_band, w, FP64 ? w.grid_fp64_band : w.grid_mixed_band);
    if (rc != STEPS_OK) return rc;
    int unused = 0;                                  // the SPLIT variants only need their shared-memory attribute set
    if constexpr (FP64) {
        rc = persistent_grid(forces_sym_kernel<SYM_FP64_THREADS, SYM_FP64_RI, false>, sym_smem_bytes(), w, w.grid_sym, SYM_FP64_THREADS);
        if (rc == STEPS_OK && !w.sym_split_ready)
            rc = persistent_grid(forces_sym_kernel<SYM_FP64_THREADS, SYM_FP64_RI, true>, sym_smem_bytes(), w, unused, SYM_FP64_THREADS);
        if (w.grid_sym > w.num_sms) w.grid_sym = w.num_sms;
    } else {
        rc = persistent_grid(forces_sym_mixed_kernel<SYM_MIXED_THREADS, SYM_MIXED_RI, false>, sym_mixed_smem_bytes<SYM_MIXED_THREADS, SYM_MIXED_RI>(),
                             w, w.grid_sym_mixed, SYM_MIXED_THREADS);
        if (rc == STEPS_OK && !w.sym_split_ready_mixed)
            rc = persistent_grid(forces_sym_mixed_kernel<SYM_MIXED_THREADS, SYM_MIXED_RI, true>, sym_mixed_smem_bytes<SYM_MIXED_THREADS, SYM_MIXED_RI>(),
                                 w, unused, SYM_MIXED_THREADS);
        if (w.grid_sym_mixed > w.num_sms) w.grid_sym_mixed = w.num_sms;      // one CTA per SM: the item shares stay equal
    }
    if (rc != STEPS_OK) return rc;
    (FP64 ? w.sym_split_ready : w.sym_split_ready_mixed) = true;
    const int P = FP64 ? w.grid_fp64_band : w.grid_mixed_band, Ps = FP64 ? w.grid_sym : w.grid_sym_mixed;
    const bool prof = g_profile.load() != 0;
    if (prof && !w.ev0) { STEPS_CUDA(cudaEventCreate(&w.ev0)); STEPS_CUDA(cudaEventCreate(&w.ev1)); }

    // Parts per item: with few blocks an item (0.3-0.7 ms) is too coarse a unit for 148 SMs, so its rounds are shared among
    // `split` sub-items (a power of two, at most the warps per CTA).
    int split = 1;
    const int max_split = (FP64 ? SYM_FP64_THREADS : SYM_MIXED_THREADS) / 32;
    if constexpr (FP64) {
        // the part count that minimises  ceil(K s / CTAs) x (1 / s + c):  the slowest CTA's parts times the cost of a part, an
        // s-th of an item plus a fixed cost c = 1/73 of an item (column copy, zeroing, 96 KiB of records: about 10 us, from
        // the measured times at N = 32,768 ... 98,304, profiles/r02_sizes.md); K estimated for a band of one block to
        // either side; whole items (the kernel variant with compile-time loop bounds) preferred by 3 %; at least the
        // 2 sub-items per CTA below which the plan gives the items up (sym_plan_finalize)
        const double Kest = (double)std::max(1ll, sym_items_max(N) - (nb - 1));
        double best = 0.0;
        for (int s = max_split; s >= 1; s /= 2) {
            if (s < max_split && Kest * s < 2.0 * Ps) break;
            const double cost = std::ceil(Kest * s / Ps) * (1.0 / s + 1.0 / 73.0) * (s == 1 ? 0.97 : 1.0);
            if (best == 0.0 || cost < best) { best = cost; split = s; }
        }
    } else if (nb < SYM_MIXED_WHOLE_ITEMS_BLOCKS) split = 4;

    prep_tiles<Tile><<<ntp, TJ, 0, st>>>(pos, mass, soft, N, tiles, &w.plan->W);
    sym_band_width<Tile><<<nb, 128, 0, st>>>(tiles, nb, w.plan);
    sym_plan_finalize<<<1, 1024, 0, st>>>(w.plan, nb, (FP64 ? 2 : 1) * Ps, split, 1);
    if (prof) STEPS_CUDA(cudaEventRecord(w.ev0, st));
    double* hi = w.acc_dd;
    double* lo = w.acc_dd + 3 * N;
    if (nb <= SYM_SPLITJ_BAND_MAX_BLOCKS && share_world == 1 && g_splitj.load() != 0) {
        // few blocks: the band's (i-block, tile) visits are too few for the ring driver (N = 32,768: 384 visits for 148 CTAs,
        // 0.28 of peak); the split-j driver takes the band instead, one 128-particle group per CTA, 64-source units
        auto sj = forces_splitj_kernel<Path, 0>;
        constexpr int smem_sj = Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double);
        static bool sj_attr_set = false;
        if (!sj_attr_set) { STEPS_CUDA(cudaFuncSetAttribute(sj, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_sj)); sj_attr_set = true; }
        const long long groups = (N + SPLITJ_GROUP - 1) / SPLITJ_GROUP;
        // the band's units of a group split over 1 or 2 CTAs, whichever makes the grid closest to whole waves (one CTA per SM;
        // more parts leave a warp less than three units: measured slower at N = 32,768)
        long long jsplit = 1;
        double best = 0.0;
        for (long long j = 1; j <= 4 && 96 / j >= 48; ++j) {       // (a band of half-width 1 is 96 units of 64 sources per group)
            const double waves = (double)(groups * j) / w.num_sms, eff = waves / std::ceil(waves);
            if (eff > best + 0.03) { best = eff; jsplit = j; }
        }
        const long long rec_cap = (long long)(partial_bytes(N) / (sizeof(double) * 6 * SPLITJ_GROUP));
        if (groups * jsplit > rec_cap) jsplit = 1;
        sj<<<dim3((unsigned)groups, (unsigned)jsplit), CTA_THREADS, smem_sj, st>>>(pos, soft, N, tiles, (int)ntiles_of(N), 64, 0, N, hi, w.partials, 0,
                                                                                     0.0, 0.0, NO_FUSE, w.plan, lo);
        g_launches += 4;
        if (jsplit > 1) {
            forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(w.partials, (int)jsplit, N, hi, NO_FUSE, lo);
            g_launches++;
        }
    } else {
        band<<<P, CTA_THREADS, smem_band, st>>>(pos, soft, N, tiles, ntp, 0, N, nb, w.partials, 0, 0.0, 0.0, w.plan, 1, share_rank, share_world);
        forces_band_reduce_kernel<Path::NOUT><<<(int)((N + 255) / 256), 256, 0, st>>>(w.partials, w.plan, P, N, acc_out, 1, hi, lo, share_rank,
                                                                                       share_world);
        g_launches += 5;
    }
    // in sub-items; a share has at most ceil(all / share_world) of them (the kernels clamp to the share's actual end)
    const long long items = w.sym_panel_items, kmax = (sym_items_max(N) * split + share_world - 1) / share_world;
    double* rowrec = w.sym_records;
    double* colrec = w.sym_records + (size_t)items * 3 * IB;
    for (long long k0 = 0; k0 < kmax; k0 += items) {
        const long long k1 = std::min(kmax, k0 + items);
        if constexpr (FP64) {
            auto k = split == 1 ? forces_sym_kernel<SYM_FP64_THREADS, SYM_FP64_RI, false> : forces_sym_kernel<SYM_FP64_THREADS, SYM_FP64_RI, true>;
            k<<<Ps, SYM_FP64_THREADS, sym_smem_bytes(), st>>>(tiles, w.plan, k0, k1, rowrec, colrec, 0, split, share_rank, share_world);
        } else {
            auto k = split == 1 ? forces_sym_mixed_kernel<SYM_MIXED_THREADS, SYM_MIXED_RI, false>
                                : forces_sym_mixed_kernel<SYM_MIXED_THREADS, SYM_MIXED_RI, true>;
            k<<<Ps, SYM_MIXED_THREADS, sym_mixed_smem_bytes<SYM_MIXED_THREADS, SYM_MIXED_RI>(), st>>>(tiles, w.plan, k0, k1, rowrec, colrec, split,
                                                                                                       share_rank, share_world);
        }
        forces_sym_reduce_kernel<<<(int)((N + 255) / 256), 256, 0, st>>>(w.plan, rowrec, colrec, k0, k1, N, hi, lo,
                                                                          k1 == kmax ? 1 : 0, acc_out, split,
                                                                          share_world == 1 ? t_fuse : NO_FUSE, share_rank, share_world);
        g_launches += 2;
    }
    if (prof) { STEPS_CUDA(cudaEventRecord(w.ev1, st)); w.ev_valid = true; }
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

// The group-ring driver has one CTA per (group, part of the tile range) and one resident CTA per SM: with fewer groups than
// SMs the tile range is split so that the grid is one wave; otherwise over 1...8 parts, whichever makes the grid closest
// to whole waves (a CTA runs for a long time -- milliseconds in the image sum -- and a ragged last wave shows).
long long boxring_jsplit(long long groups, long long nt, long long N, const Workspace& w)
{
    long long jsplit = 1;
    if (groups < w.num_sms) {
        jsplit = w.num_sms / groups;
    } else {
        double best = 0.0;
        for (long long j = 1; j <= 8; ++j) {
            const double waves = (double)(groups * j) / w.num_sms;
            const double eff = waves / std::ceil(waves);
            if (eff > best + 0.02) { best = eff; jsplit = j; }
        }
    }
    jsplit = std::max(1ll, std::min(jsplit, nt / BOXRING_G));                 // at least one tile per sub-ring
    const long long rec_cap = (long long)(partial_bytes(N) / (sizeof(double) * 6 * SPLITJ_GROUP));
    if (groups * jsplit > rec_cap) jsplit = std::max(1ll, rec_cap / groups);
    return jsplit;
}

// Split-j driver (force_driver.cuh): one 128-particle group per CTA column, the j-range split over the warps and over
// `jsplit` CTAs.  The source sub-range per work unit shrinks (256 -> 64) until there are about two units per resident warp.
template <typename Path, int BOX>
int launch_splitj(const double* pos, const double* soft, long long N, const typename Path::Tile* tiles, int nt,
                  long long i_begin, long long i_end, double* acc_out, cudaStream_t st, Workspace& w, double L)
{
    const long long cnt = i_end - i_begin;
    const long long groups = (cnt + SPLITJ_GROUP - 1) / SPLITJ_GROUP;
    const long long warps = (long long)w.num_sms * (CTA_THREADS / 32);
    int sub = TJ;
    while (sub > 64 && groups * nt * (TJ / sub) < 4 * warps) sub /= 2;
    const long long units = (long long)nt * (TJ / sub);                      // per group
    // one CTA per SM is resident (512 threads, up to 96 KiB of accumulators): with fewer groups than SMs the j-range is split
    // over floor(SMs / groups) CTAs so that the whole grid is ONE wave; with more groups than SMs there is nothing to split
    long long jsplit = groups < w.num_sms ? w.num_sms / groups : 1;
    // ... or over up to 8 CTAs in several waves, when that fills the SMs better and leaves each CTA >= 2^24 pairs (~20 us)
    {
        const double one = (double)(groups * jsplit) / w.num_sms;
        double best = one / std::ceil(one);
        for (long long j = jsplit + 1; j <= 8; ++j) {
            if ((double)SPLITJ_GROUP * (double)N / (double)j < 16777216.0) break;
            const double waves = (double)(groups * j) / w.num_sms, eff = waves / std::ceil(waves);
            if (eff > best + 0.05) { best = eff; jsplit = j; }
        }
    }
    jsplit = std::max(1ll, std::min(jsplit, units / (CTA_THREADS / 32)));
    const long long rec_cap = (long long)(partial_bytes(N) / (sizeof(double) * 6 * SPLITJ_GROUP));
    if (groups * jsplit > rec_cap) jsplit = std::max(1ll, rec_cap / groups);
    if (groups > 0x7fffffffll || jsplit > 65535) return STEPS_EINVAL;
    auto kern = forces_splitj_kernel<Path, BOX>;
    constexpr int smem = Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double);
    static bool attr_set = false;                                                // per instantiation
    if (!attr_set) { STEPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); attr_set = true; }
    const bool prof = g_profile.load() != 0;
    if (prof) {
        if (!w.ev0) { STEPS_CUDA(cudaEventCreate(&w.ev0)); STEPS_CUDA(cudaEventCreate(&w.ev1)); }
        STEPS_CUDA(cudaEventRecord(w.ev0, st));
    }
    const Eq12Fuse fuse = (BOX == 0 && i_begin == 0 && i_end == N) ? t_fuse : NO_FUSE;
    kern<<<dim3((unsigned)groups, (unsigned)jsplit), CTA_THREADS, smem, st>>>(pos, soft, N, tiles, nt, sub, i_begin, i_end, acc_out,
                                                                                w.partials, 0, L, L > 0.0 ? 1.0 / L : 0.0, fuse, nullptr, nullptr);
    g_launches++;
    if (jsplit > 1) {
        forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(w.partials, (int)jsplit, cnt, acc_out, fuse);
        g_launches++;
    }
    if (prof) { STEPS_CUDA(cudaEventRecord(w.ev1, st)); w.ev_valid = true; }
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

// The ring driver's (i-block, j-tile) items are too few to fill the SMs below this many per SM: split-j driver instead,
// as long as its groups fit one wave of CTAs (N <= 128 x SMs = 18,944 on B200; measured 3.7x at N = 4,096).
inline bool use_splitj(long long cnt, long long N, const Workspace& w)
{
    return g_splitj.load() != 0 && (cnt + SPLITJ_GROUP - 1) / SPLITJ_GROUP <= w.num_sms && nblocks_of(cnt) * ntiles_of(N) < 8ll * w.num_sms;
}

// block_stride == 1: forces on [i_begin, i_end).  block_stride > 1 (steps_forces_blocks): forces on the blocks
// i_begin / IB + k block_stride, k = 0, 1, ...; i_end = N; `cnt` = how many particles that is; acc_out packed over them.
template <typename Path>
int launch_forces(const double* pos, const double* mass, const double* soft, long long N, long long i_begin,
                  long long i_end, double* acc_out, cudaStream_t st, Workspace& w, int& grid_cache, int block_stride = 1,
                  long long cnt_strided = 0)
{
    using Tile = typename Path::Tile;
    if (block_stride == 1 && i_begin == 0 && i_end == N && g_driver.load() == 0 && sym_eligible(N, Path::NOUT == 3) && w.sym_records &&
        (Path::NOUT == 6 || g_sym_enabled.load() != 2))      // "sym" = 2: fp64 path only
        return launch_forces_sym<Path>(pos, mass, soft, N, acc_out, st, w);
    const int nt = (int)ntiles_of(N);
    Tile* tiles = reinterpret_cast<Tile*>(w.tiles);
    prep_tiles<Tile><<<nt, TJ, 0, st>>>(pos, mass, soft, N, tiles, nullptr);
    g_launches++;
    const long long cnt = block_stride == 1 ? i_end - i_begin : cnt_strided;
    const int nb = (int)nblocks_of(cnt);
    if (block_stride == 1 && g_driver.load() == 0 && use_splitj(cnt, N, w))
        return launch_splitj<Path, 0>(pos, soft, N, tiles, nt, i_begin, i_end, acc_out, st, w, 0.0);
    if (g_driver.load() == 1 && block_stride == 1) {
        const int smem = stage_stride((int)sizeof(Tile)) + Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double);
        STEPS_CUDA(cudaFuncSetAttribute(forces_v1_kernel<Path>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        forces_v1_kernel<Path><<<nb, CTA_THREADS, smem, st>>>(pos, soft, N, tiles, nt, i_begin, i_end, acc_out, 0);
        g_launches++;
    } else {
        constexpr int smem = persistent_smem_bytes<Path, STAGES>();
        auto kern = forces_persistent_kernel<Path, STAGES>;
        const int rc = persistent_grid(kern, smem, w, grid_cache);
        if (rc != STEPS_OK) return rc;
        const int P = grid_cache;
        const bool prof = g_profile.load() != 0;
        if (prof) {
            if (!w.ev0) { STEPS_CUDA(cudaEventCreate(&w.ev0)); STEPS_CUDA(cudaEventCreate(&w.ev1)); }
            STEPS_CUDA(cudaEventRecord(w.ev0, st));
        }
        kern<<<P, CTA_THREADS, smem, st>>>(pos, soft, N, tiles, nt, i_begin, i_end, nb, w.partials, 0, 0.0, 0.0, nullptr, block_stride, 0, 1);
        if (prof) { STEPS_CUDA(cudaEventRecord(w.ev1, st)); w.ev_valid = true; }
        forces_reduce_kernel<Path::NOUT><<<(int)((cnt + 255) / 256), 256, 0, st>>>(
            w.partials, nt, nb, P, cnt, acc_out, (block_stride == 1 && i_begin == 0 && i_end == N) ? t_fuse : NO_FUSE);
        g_launches += 2;
    }
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

int forces_impl(const double* pos, const double* mass, const double* soft, long long N, long long i_begin,
                long long i_end, double* acc_out, int mixed, steps_stream_t stream)
{
    if (!pos || !mass || !soft || !acc_out || N < 1) return STEPS_EINVAL;
    if (i_begin < 0 || i_end > N || i_begin >= i_end) return STEPS_EINVAL;
    if (N > (1ll << 31) - IB) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(mass) || misaligned(soft) || misaligned(acc_out)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = ensure_workspace(dev, N, st);
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    rc = claim_scratch(w, st);
    if (rc != STEPS_OK) return rc;
    rc = mixed ? launch_forces<MixedPath>(pos, mass, soft, N, i_begin, i_end, acc_out, st, w, w.grid_mixed)
               : launch_forces<Fp64Path>(pos, mass, soft, N, i_begin, i_end, acc_out, st, w, w.grid_fp64);
    if (rc != STEPS_OK) return rc;
    return release_scratch(w, st);
}

// Leading-image periodic box (steps_forces_quasi_periodic).  One 128-particle group per CTA column (forces_boxring_kernel);
// from 9 (fp64) / 80 (mixed) blocks the far pairs of DIFFERENT blocks go through the pair-symmetric kernels
// (forces_sym_box_kernel / forces_sym_mixed_box_kernel), each evaluated once, and the group-ring kernel runs in restricted
// mode (the groups' own blocks + the units that may hold a softened pair).  All decisions that depend on the data are taken
// on the device (pair_decision on the group boxes; the plan falls back to "everything one-sided" when the items are too few).
template <typename Path>
int launch_forces_box(const double* pos, const double* mass, const double* soft, long long N, double L, double* acc_out,
                      cudaStream_t st, Workspace& w)
{
    using Tile = typename Path::Tile;
    constexpr bool FP64 = Path::NOUT == 6;
    const int nb = (int)nblocks_of(N);
    const int nt = (int)ntiles_of(N);
    Tile* tiles = reinterpret_cast<Tile*>(w.tiles);
    const bool sym = g_driver.load() == 0 && sym_eligible(N, !FP64) && nb >= (FP64 ? SYM_BOX_MIN_BLOCKS : SYM_BOX_MIN_BLOCKS_MIXED) && w.sym_records &&
                     (FP64 || g_sym_enabled.load() != 2);
    const long long groups = (N + SPLITJ_GROUP - 1) / SPLITJ_GROUP;
    const long long jsplit = boxring_jsplit(groups, nt, N, w);
    if (groups > 0x7fffffffll || jsplit > 65535) return STEPS_EINVAL;
    auto ring = forces_boxring_kernel<Path, 1>;
    constexpr int smem = boxring_smem_bytes<Path, 1>();
    static bool attr_set = false;                                              // per instantiation
    if (!attr_set) { STEPS_CUDA(cudaFuncSetAttribute(ring, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); attr_set = true; }
    const bool prof = g_profile.load() != 0;
    if (prof && !w.ev0) { STEPS_CUDA(cudaEventCreate(&w.ev0)); STEPS_CUDA(cudaEventCreate(&w.ev1)); }
    const dim3 grid((unsigned)groups, (unsigned)jsplit);

    if (!sym) {
        prep_tiles<Tile><<<nt, TJ, 0, st>>>(pos, mass, soft, N, tiles, nullptr);
        if (prof) STEPS_CUDA(cudaEventRecord(w.ev0, st));
        ring<<<grid, CTA_THREADS, smem, st>>>(pos, soft, N, tiles, nt, acc_out, w.partials, 0, L, 1.0 / L, nullptr, nullptr, nullptr);
        g_launches += 2;
        if (jsplit > 1) {
            forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(w.partials, (int)jsplit, N, acc_out, NO_FUSE);
            g_launches++;
        }
        if (prof) { STEPS_CUDA(cudaEventRecord(w.ev1, st)); w.ev_valid = true; }
        STEPS_CUDA(cudaGetLastError());
        return STEPS_OK;
    }

    const int ntp = nb * TPB, ngm = nb * (IB / SPLITJ_GROUP);
    int Ps = 0;
    int split = 1;
    if constexpr (FP64) {
        static int grid_box = 0, unused = 0;
        int rc = persistent_grid(forces_sym_box_kernel<SYM_FP64_THREADS, SYM_FP64_RI, false>, sym_box_smem_bytes(), w, grid_box, SYM_FP64_THREADS);
        if (rc == STEPS_OK && unused == 0)
            rc = persistent_grid(forces_sym_box_kernel<SYM_FP64_THREADS, SYM_FP64_RI, true>, sym_box_smem_bytes(), w, unused, SYM_FP64_THREADS);
        if (rc != STEPS_OK) return rc;
        Ps = std::min(grid_box, w.num_sms);
        while (split < SYM_FP64_THREADS / 32 && sym_items_max(N) * split < 24ll * Ps) split *= 2;
    } else {
        static int grid_box = 0;
        const int rc = persistent_grid(forces_sym_mixed_box_kernel<SYM_MIXED_THREADS, SYM_MIXED_RI, false>,
                                       sym_mixed_box_smem_bytes<SYM_MIXED_THREADS, SYM_MIXED_RI>(), w, grid_box, SYM_MIXED_THREADS);
        if (rc != STEPS_OK) return rc;
        Ps = std::min(grid_box, w.num_sms);
    }
    prep_tiles<Tile><<<ntp, TJ, 0, st>>>(pos, mass, soft, N, tiles, &w.plan->W);          // W = 0: every block pair is an item
    group_meta_kernel<Tile><<<(ngm + 3) / 4, 128, 0, st>>>(pos, soft, N, tiles, w.gm, ngm);
    sym_plan_finalize<<<1, 1024, 0, st>>>(w.plan, nb, 2 * Ps, split, 0);
    if (prof) STEPS_CUDA(cudaEventRecord(w.ev0, st));
    double* hi = w.acc_dd;
    double* lo = w.acc_dd + 3 * N;
    // one-sided part: the possibly-softened units of other blocks (zero if the plan kept no items), then the groups' own
    // blocks (everything if the plan kept no items) added to it; groups >= SMs here, so the tile range is never split
    auto gen = forces_boxgen_kernel<Path>;
    static bool gen_attr_set = false;
    if (!gen_attr_set) { STEPS_CUDA(cudaFuncSetAttribute(gen, cudaFuncAttributeMaxDynamicSharedMemorySize, boxgen_smem_bytes<Path>())); gen_attr_set = true; }
    // (the unit range of a group is split over up to 8 CTAs, see forces_boxgen_kernel; their records use the symmetric
    // kernels' record buffer, which is free until the first panel)
    long long gsplit = std::max(1, g_box_gsplit.load());
    while (gsplit > 1 && (size_t)groups * gsplit * 6 * SPLITJ_GROUP * sizeof(double) > sym_record_bytes(w.sym_panel_items)) gsplit /= 2;
    gen<<<dim3((unsigned)groups, (unsigned)gsplit), CTA_THREADS, boxgen_smem_bytes<Path>(), st>>>(pos, soft, N, tiles, nt, hi, lo, w.sym_records,
                                                                                                   L, 1.0 / L, w.gm, w.plan);
    if (gsplit > 1) {
        forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(w.sym_records, (int)gsplit, N, hi, NO_FUSE, lo);
        g_launches++;
    }
    ring<<<(unsigned)groups, CTA_THREADS, smem, st>>>(pos, soft, N, tiles, nt, hi, w.partials, 0, L, 1.0 / L, w.gm, w.plan, lo);
    g_launches += 5;
    const long long items = w.sym_panel_items, kmax = sym_items_max(N) * split;          // in sub-items
    double* rowrec = w.sym_records;
    double* colrec = w.sym_records + (size_t)items * 3 * IB;
    for (long long k0 = 0; k0 < kmax; k0 += items) {
        const long long k1 = std::min(kmax, k0 + items);
        if constexpr (FP64) {
            auto k = split == 1 ? forces_sym_box_kernel<SYM_FP64_THREADS, SYM_FP64_RI, false> : forces_sym_box_kernel<SYM_FP64_THREADS, SYM_FP64_RI, true>;
            k<<<Ps, SYM_FP64_THREADS, sym_box_smem_bytes(), st>>>(tiles, w.plan, w.gm, k0, k1, rowrec, colrec, 0, split, L, 1.0 / L);
        } else {
            forces_sym_mixed_box_kernel<SYM_MIXED_THREADS, SYM_MIXED_RI, false>
                <<<Ps, SYM_MIXED_THREADS, sym_mixed_box_smem_bytes<SYM_MIXED_THREADS, SYM_MIXED_RI>(), st>>>(tiles, w.plan, w.gm, k0, k1, rowrec,
                                                                                                               colrec, split, L, 1.0 / L);
        }
        forces_sym_reduce_kernel<<<(int)((N + 255) / 256), 256, 0, st>>>(w.plan, rowrec, colrec, k0, k1, N, hi, lo,
                                                                          k1 == kmax ? 1 : 0, acc_out, split, NO_FUSE);
        g_launches += 2;
    }
    if (prof) { STEPS_CUDA(cudaEventRecord(w.ev1, st)); w.ev_valid = true; }
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

// Image sum (steps_forces_periodic) from 9 blocks: every far meeting of two groups of different blocks ONCE
// (forces_sym_img_kernel: the image sum of a pair is antisymmetric), the possibly-softened units by
// forces_boxgen_kernel<Fp64Path, 2>, the groups' own blocks by the group-ring kernel in restricted mode.
int launch_forces_images_sym(const double* pos, const double* mass, const double* soft, long long N, double L, double* acc_out,
                             cudaStream_t st, Workspace& w)
{
    using Path = Fp64Path;
    using Tile = Path::Tile;
    const int nb = (int)nblocks_of(N), nt = (int)ntiles_of(N);
    const int ntp = nb * TPB, ngm = nb * (IB / SPLITJ_GROUP);
    Tile* tiles = reinterpret_cast<Tile*>(w.tiles);
    const long long groups = (N + SPLITJ_GROUP - 1) / SPLITJ_GROUP;
    if (groups > 0x7fffffffll) return STEPS_EINVAL;
    static int grid_img = 0, unused = 0;
    int rc = persistent_grid(forces_sym_img_kernel<SYM_FP64_THREADS, SYM_FP64_RI, false>, sym_img_smem_bytes(), w, grid_img, SYM_FP64_THREADS);
    if (rc == STEPS_OK && unused == 0)
        rc = persistent_grid(forces_sym_img_kernel<SYM_FP64_THREADS, SYM_FP64_RI, true>, sym_img_smem_bytes(), w, unused, SYM_FP64_THREADS);
    if (rc != STEPS_OK) return rc;
    const int Ps = std::min(grid_img, w.num_sms);
    int split = 1;
    while (split < SYM_FP64_THREADS / 32 && sym_items_max(N) * split < 24ll * Ps) split *= 2;
    auto gen = forces_boxgen_kernel<Path, 2>;
    static bool attr_set = false;
    if (!attr_set) {
        STEPS_CUDA(cudaFuncSetAttribute(gen, cudaFuncAttributeMaxDynamicSharedMemorySize, boxgen_smem_bytes<Path>()));
        attr_set = true;
    }
    prep_tiles<Tile><<<ntp, TJ, 0, st>>>(pos, mass, soft, N, tiles, &w.plan->W);          // W = 0: every block pair is an item
    group_meta_kernel<Tile><<<(ngm + 3) / 4, 128, 0, st>>>(pos, soft, N, tiles, w.gm, ngm);
    sym_plan_finalize<<<1, 1024, 0, st>>>(w.plan, nb, 0, split, 0);                      // (no minimum: this route has no one-sided fallback kernel)
    double* hi = w.acc_dd;
    double* lo = w.acc_dd + 3 * N;
    long long gsplit = std::max(1, g_box_gsplit.load());
    while (gsplit > 1 && (size_t)groups * gsplit * 6 * SPLITJ_GROUP * sizeof(double) > sym_record_bytes(w.sym_panel_items)) gsplit /= 2;
    gen<<<dim3((unsigned)groups, (unsigned)gsplit), CTA_THREADS, boxgen_smem_bytes<Path>(), st>>>(pos, soft, N, tiles, nt, hi, lo, w.sym_records,
                                                                                                   L, 1.0 / L, w.gm, w.plan);
    if (gsplit > 1) {
        forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(w.sym_records, (int)gsplit, N, hi, NO_FUSE, lo);
        g_launches++;
    }
    g_launches += 4;
    const long long items = w.sym_panel_items, kmax = sym_items_max(N) * split;
    double* rowrec = w.sym_records;
    double* colrec = w.sym_records + (size_t)items * 3 * IB;
    auto k = split == 1 ? forces_sym_img_kernel<SYM_FP64_THREADS, SYM_FP64_RI, false> : forces_sym_img_kernel<SYM_FP64_THREADS, SYM_FP64_RI, true>;
    // the blocks themselves (diagonal items: every pair of groups of a block once), then the block pairs, panel by panel
    if ((long long)nb * split <= items) {
        k<<<Ps, SYM_FP64_THREADS, sym_img_smem_bytes(), st>>>(tiles, w.plan, w.gm, 0, (long long)nb * split, rowrec, colrec, split, L, 1.0 / L, 1);
        forces_sym_diag_reduce<<<(int)((N + 255) / 256), 256, 0, st>>>(w.plan, rowrec, colrec, split, N, hi, lo);
        g_launches += 2;
    } else {
        return STEPS_EINVAL;                         // (sym_panel_items set below the number of blocks)
    }
    for (long long k0 = 0; k0 < kmax; k0 += items) {
        const long long k1 = std::min(kmax, k0 + items);
        k<<<Ps, SYM_FP64_THREADS, sym_img_smem_bytes(), st>>>(tiles, w.plan, w.gm, k0, k1, rowrec, colrec, split, L, 1.0 / L, 0);
        forces_sym_reduce_kernel<<<(int)((N + 255) / 256), 256, 0, st>>>(w.plan, rowrec, colrec, k0, k1, N, hi, lo, k1 == kmax ? 1 : 0, acc_out,
                                                                          split, NO_FUSE);
        g_launches += 2;
    }
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

template <typename Path, int BOX>
int launch_forces_periodic(const double* pos, const double* mass, const double* soft, long long N, double L, double* acc_out,
                           cudaStream_t st, Workspace& w)
{
    using Tile = typename Path::Tile;
    const int nt = (int)ntiles_of(N);
    Tile* tiles = reinterpret_cast<Tile*>(w.tiles);
    int rc = claim_scratch(w, st);
    if (rc != STEPS_OK) return rc;
    if constexpr (BOX == 1) {
        rc = launch_forces_box<Path>(pos, mass, soft, N, L, acc_out, st, w);
        if (rc != STEPS_OK) return rc;
        return release_scratch(w, st);
    } else {
        if (g_driver.load() == 0 && sym_eligible(N, false) && nblocks_of(N) >= SYM_BOX_MIN_BLOCKS && w.sym_records) {
            rc = launch_forces_images_sym(pos, mass, soft, N, L, acc_out, st, w);
            if (rc != STEPS_OK) return rc;
            return release_scratch(w, st);
        }
        // Image sum: the group-ring driver with BOX = 2.  The tile range is split over `jsplit` CTAs so that the grid is
        // (close to) whole waves of one CTA per SM -- an image-sum CTA runs for milliseconds, a ragged last wave shows.
        prep_tiles<Tile><<<nt, TJ, 0, st>>>(pos, mass, soft, N, tiles, nullptr);
        g_launches++;
        const long long groups = (N + SPLITJ_GROUP - 1) / SPLITJ_GROUP;
        const long long jsplit = boxring_jsplit(groups, nt, N, w);
        if (groups > 0x7fffffffll) return STEPS_EINVAL;
        auto kern = forces_boxring_kernel<Path, 2>;
        constexpr int smem = boxring_smem_bytes<Path, 2>();
        static bool attr_set = false;
        if (!attr_set) { STEPS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); attr_set = true; }
        kern<<<dim3((unsigned)groups, (unsigned)jsplit), CTA_THREADS, smem, st>>>(pos, soft, N, tiles, nt, acc_out, w.partials, 0, L, 1.0 / L,
                                                                                    nullptr, nullptr, nullptr);
        g_launches++;
        if (jsplit > 1) {
            forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(w.partials, (int)jsplit, N, acc_out, NO_FUSE);
            g_launches++;
        }
        STEPS_CUDA(cudaGetLastError());
        return release_scratch(w, st);
    }
}

}  // namespace

// ---- steps_forces_static: the fp64 split-j evaluation with its scratch in a file-scope device array (include/steps.h) ----
// [ STATIC_TILES tile records | STATIC_RECORDS split-j partial records of 6 x 128 doubles ].  In HOST code the array's name
// is a host-side stand-in, not a device address: static_scratch_of() asks the runtime for the address once per device.
constexpr int STATIC_TILES = STEPS_STATIC_MAX_N / TJ;                        // 64
constexpr int STATIC_RECORDS = 256;                                          // >= groups x jsplit (<= SMs of the device)
constexpr size_t STATIC_TILE_BYTES = sizeof(TileF64) * STATIC_TILES;
constexpr size_t STATIC_RECORD_BYTES = sizeof(double) * 6 * SPLITJ_GROUP;
static_assert(STEPS_STATIC_MAX_N % TJ == 0 && STATIC_TILE_BYTES % 256 == 0, "the records start on a 256 B boundary");
static_assert(STATIC_TILE_BYTES + STATIC_RECORD_BYTES * STATIC_RECORDS == STEPS_STATIC_SCRATCH_BYTES, "include/steps.h states the size");
static __device__ __align__(256) unsigned char g_static_scratch[STEPS_STATIC_SCRATCH_BYTES];

namespace {

struct StaticState {
    unsigned char* scratch = nullptr;   // device address of g_static_scratch on this device
    int num_sms = 0;
    bool ready = false;
};
StaticState g_static[MAX_DEVICES];
std::mutex g_static_mutex;

// Once per device, with that device current: the array's device address, the SM count, the kernel's shared-memory opt-in.
// Nothing here allocates device memory.
int static_scratch_of(int dev, StaticState** out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticState& s = g_static[dev];
    if (!s.ready) {
        void* ptr = nullptr;
        STEPS_CUDA(cudaGetSymbolAddress(&ptr, g_static_scratch));
        if (ptr == nullptr) return STEPS_ECUDA;
        STEPS_CUDA(cudaDeviceGetAttribute(&s.num_sms, cudaDevAttrMultiProcessorCount, dev));
        constexpr int smem = Fp64Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double);
        STEPS_CUDA(cudaFuncSetAttribute(forces_splitj_kernel<Fp64Path, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        s.scratch = static_cast<unsigned char*>(ptr);
        s.ready = true;
    }
    *out = &s;
    return STEPS_OK;
}

}  // namespace

extern "C" {

int steps_forces_quasi_periodic(const double* pos, const double* mass, const double* soft, long long N, double L,
                                double* acc, int mixed, steps_stream_t stream)
{
    if (!pos || !mass || !soft || !acc || N < 1 || !(L > 0.0)) return STEPS_EINVAL;
    if (N > (1ll << 31) - IB) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(mass) || misaligned(soft) || misaligned(acc)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, N, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Workspace& w = g_ws[dev];
    return mixed ? launch_forces_periodic<MixedPath, 1>(pos, mass, soft, N, L, acc, st, w)
                 : launch_forces_periodic<Fp64Path, 1>(pos, mass, soft, N, L, acc, st, w);
}

int steps_forces_periodic(const double* pos, const double* mass, const double* soft, long long N, double L, double* acc,
                          steps_stream_t stream)
{
    if (!pos || !mass || !soft || !acc || N < 1 || !(L > 0.0)) return STEPS_EINVAL;
    if (N > (1ll << 31) - IB) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(mass) || misaligned(soft) || misaligned(acc)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, N, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    return launch_forces_periodic<Fp64Path, 2>(pos, mass, soft, N, L, acc, reinterpret_cast<cudaStream_t>(stream), w);
}

int steps_forces(const double* pos, const double* mass, const double* soft, long long N, double* acc,
                 steps_stream_t stream)
{
    return forces_impl(pos, mass, soft, N, 0, N, acc, 0, stream);
}

int steps_forces_mixed(const double* pos, const double* mass, const double* soft, long long N, double* acc,
                       steps_stream_t stream)
{
    return forces_impl(pos, mass, soft, N, 0, N, acc, 1, stream);
}

int steps_forces_static(const double* pos, const double* mass, const double* soft, long long N, double* acc,
                        steps_stream_t stream)
{
    if (!pos || !mass || !soft || !acc || N < 1) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(mass) || misaligned(soft) || misaligned(acc)) return STEPS_EINVAL;
    if (N > STEPS_STATIC_MAX_N) return STEPS_ETOOLARGE;
    int dev;
    int rc = current_device(&dev);                       // (device query only: sm_100 or STEPS_EUNSUPPORTED)
    if (rc != STEPS_OK) return rc;
    StaticState* s = nullptr;
    rc = static_scratch_of(dev, &s);
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    TileF64* tiles = reinterpret_cast<TileF64*>(s->scratch);
    double* records = reinterpret_cast<double*>(s->scratch + STATIC_TILE_BYTES);

    // the launch shape of launch_splitj<Fp64Path, 0> at this N (one wave: groups x jsplit <= SMs), so the result is
    // steps_forces' at the same N
    const int nt = (int)ntiles_of(N);
    const long long groups = (N + SPLITJ_GROUP - 1) / SPLITJ_GROUP;
    const long long warps = (long long)s->num_sms * (CTA_THREADS / 32);
    int sub = TJ;
    while (sub > 64 && groups * nt * (TJ / sub) < 4 * warps) sub /= 2;
    const long long units = (long long)nt * (TJ / sub);
    long long jsplit = groups < s->num_sms ? s->num_sms / groups : 1;
    jsplit = std::max(1ll, std::min(jsplit, units / (CTA_THREADS / 32)));
    if (groups * jsplit > STATIC_RECORDS) jsplit = std::max(1ll, STATIC_RECORDS / groups);
    constexpr int smem = Fp64Path::NOUT * R_I * CTA_THREADS * (int)sizeof(double);

    prep_tiles<TileF64><<<nt, TJ, 0, st>>>(pos, mass, soft, N, tiles, nullptr);
    forces_splitj_kernel<Fp64Path, 0><<<dim3((unsigned)groups, (unsigned)jsplit), CTA_THREADS, smem, st>>>(
        pos, soft, N, tiles, nt, sub, 0, N, acc, records, 0, 0.0, 0.0, NO_FUSE, nullptr, nullptr);
    g_launches += 2;
    if (jsplit > 1) {
        forces_splitj_reduce<<<(unsigned)groups, SPLITJ_GROUP, 0, st>>>(records, (int)jsplit, N, acc, NO_FUSE);
        g_launches++;
    }
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

int steps_forces_range(const double* pos, const double* mass, const double* soft, long long N, long long i_begin,
                       long long i_end, double* acc_out, int mixed, steps_stream_t stream)
{
    return forces_impl(pos, mass, soft, N, i_begin, i_end, acc_out, mixed, stream);
}

int steps_block_size(void) { return IB; }

int steps_forces_blocks(const double* pos, const double* mass, const double* soft, long long N, long long first_block,
                        long long block_stride, double* acc_out, int mixed, steps_stream_t stream)
{
    if (!pos || !mass || !soft || !acc_out || N < 1) return STEPS_EINVAL;
    const long long nb_all = nblocks_of(N);
    if (first_block < 0 || first_block >= nb_all || block_stride < 1 || block_stride > 0x7fffffff) return STEPS_EINVAL;
    if (N > (1ll << 31) - IB) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(mass) || misaligned(soft) || misaligned(acc_out)) return STEPS_EINVAL;
    const long long owned = (nb_all - 1 - first_block) / block_stride + 1;                     // blocks first, first + stride, ...
    const long long last = first_block + (owned - 1) * block_stride;
    const long long cnt = (owned - 1) * IB + std::min<long long>(IB, N - last * IB);
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = ensure_workspace(dev, N, st);
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    rc = claim_scratch(w, st);
    if (rc != STEPS_OK) return rc;
    rc = mixed ? launch_forces<MixedPath>(pos, mass, soft, N, first_block * IB, N, acc_out, st, w, w.grid_mixed, (int)block_stride, cnt)
               : launch_forces<Fp64Path>(pos, mass, soft, N, first_block * IB, N, acc_out, st, w, w.grid_fp64, (int)block_stride, cnt);
    if (rc != STEPS_OK) return rc;
    return release_scratch(w, st);
}

int steps_forces_share(const double* pos, const double* mass, const double* soft, long long N, int rank, int world,
                       double* acc_part, int mixed, steps_stream_t stream)
{
    if (!pos || !mass || !soft || !acc_part || N < 1 || world < 1 || rank < 0 || rank >= world) return STEPS_EINVAL;
    if (N > (1ll << 31) - IB) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(mass) || misaligned(soft) || misaligned(acc_part)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = ensure_workspace(dev, N, st);
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    const bool sym = g_driver.load() == 0 && sym_eligible(N, mixed != 0) && w.sym_records && (!mixed || g_sym_enabled.load() != 2);
    if (!sym) {                                       // too small to share (under a millisecond): rank 0 evaluates it all
        if (rank == 0) return forces_impl(pos, mass, soft, N, 0, N, acc_part, mixed, stream);
        STEPS_CUDA(cudaMemsetAsync(acc_part, 0, sizeof(double) * 3 * (size_t)N, st));
        return STEPS_OK;
    }
    rc = claim_scratch(w, st);
    if (rc != STEPS_OK) return rc;
    rc = mixed ? launch_forces_sym<MixedPath>(pos, mass, soft, N, acc_part, st, w, rank, world)
               : launch_forces_sym<Fp64Path>(pos, mass, soft, N, acc_part, st, w, rank, world);
    if (rc != STEPS_OK) return rc;
    return release_scratch(w, st);
}

int steps_forces_host(const double* pos_host, const double* mass_host, const double* soft_host, long long N,
                      double* acc_host, int mixed, steps_stream_t stream)
{
    if (!pos_host || !mass_host || !soft_host || !acc_host || N < 1) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (N > w.h_cap) {
            cudaFree(w.h_pos); cudaFree(w.h_mass); cudaFree(w.h_soft); cudaFree(w.h_acc);
            w.h_pos = w.h_mass = w.h_soft = w.h_acc = nullptr; w.h_cap = 0;
            if (cudaMalloc(&w.h_pos, sizeof(double) * 3 * N) != cudaSuccess ||
                cudaMalloc(&w.h_mass, sizeof(double) * N) != cudaSuccess ||
                cudaMalloc(&w.h_soft, sizeof(double) * N) != cudaSuccess ||
                cudaMalloc(&w.h_acc, sizeof(double) * 3 * N) != cudaSuccess) {
                cudaGetLastError();
                return STEPS_ENOMEM;
            }
            w.h_cap = N;
        }
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    STEPS_CUDA(cudaMemcpyAsync(w.h_pos, pos_host, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, st));
    STEPS_CUDA(cudaMemcpyAsync(w.h_mass, mass_host, sizeof(double) * N, cudaMemcpyHostToDevice, st));
    STEPS_CUDA(cudaMemcpyAsync(w.h_soft, soft_host, sizeof(double) * N, cudaMemcpyHostToDevice, st));
    rc = forces_impl(w.h_pos, w.h_mass, w.h_soft, N, 0, N, w.h_acc, mixed, stream);
    if (rc != STEPS_OK) return rc;
    STEPS_CUDA(cudaMemcpyAsync(acc_host, w.h_acc, sizeof(double) * 3 * N, cudaMemcpyDeviceToHost, st));
    STEPS_CUDA(cudaStreamSynchronize(st));
    return STEPS_OK;
}

int steps_kick_drift(double* pos, double* vel, const double* acc, long long N, const steps_kdk_coeffs* c,
                     steps_stream_t stream)
{
    if (!pos || !vel || !acc || !c || N < 1) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(vel) || misaligned(acc)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    KdkScalars k{c->alpha_close, c->beta_close, c->alpha_open, c->beta_open, c->gamma, c->B};
    const long long M = 3 * N;
    long long blocks = (M + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    kick_drift_kernel<<<(int)blocks, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(pos, vel, acc, M, k);
    g_launches++;
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

int steps_kdk_step(double* pos, double* vel, double* acc, const double* mass, const double* soft, long long N,
                   const steps_kdk_coeffs* c, steps_stream_t stream)
{
    if (!mass || !soft) return STEPS_EINVAL;
    int rc = steps_kick_drift(pos, vel, acc, N, c, stream);
    if (rc != STEPS_OK) return rc;
    return forces_impl(pos, mass, soft, N, 0, N, acc, c->mixed, stream);
}

int steps_kdk_step_adaptive(double* pos, double* vel, double* acc, const double* mass, const double* soft, long long N,
                            double* state5, const steps_cosmology* c, double G, double B, double eps, double dt_max,
                            int mixed, steps_stream_t stream)
{
    if (!pos || !vel || !acc || !mass || !soft || !state5 || !c || N < 1) return STEPS_EINVAL;
    if (!(eps > 0.0) || !(dt_max > 0.0)) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(vel) || misaligned(acc)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, N, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = claim_scratch(g_ws[dev], st);                      // released by the force evaluation at the end of this call
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    double* partial = w.mom_partial;
    double* coef6 = partial + 2 * MOM_BLOCKS;
    unsigned long long* fused_bits = reinterpret_cast<unsigned long long*>(partial + 2 * MOM_BLOCKS + 8);
    RunState* rs = reinterpret_cast<RunState*>(state5);
    const CosmoScalars cs{c->H0, c->Omega_m, c->Omega_r, c->Omega_L, c->Omega_k};
    // Eq. 12: the minimum over the particles was folded into `fused_bits` by the force evaluation of the PREVIOUS call of this
    // function when that call was the last thing this library launched and it was for the same arrays and parameters (the
    // candidates depend on pos, acc, soft, |G|, B, eps and on the run state's a); otherwise the O(N) pass forms it now.
    const FuseToken now{pos, acc, soft, state5, N, std::fabs(G), B, eps, g_launches.load()};
    const bool fused = w.fuse_valid && w.fuse_token == now;
    if (!fused) {
        timestep_state_stage1<<<MOM_BLOCKS, 256, 0, st>>>(pos, acc, soft, N, rs, std::fabs(G), B, eps, dt_max, partial);
        g_launches++;
    }
    step_coefficients_kernel<<<1, 32, 0, st>>>(partial, MOM_BLOCKS, rs, cs, G, B, coef6, fused ? fused_bits : nullptr, dt_max);
    const long long M = 3 * N;
    long long blocks = (M + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    kick_drift_dev_kernel<<<(int)blocks, 256, 0, st>>>(pos, vel, acc, M, coef6);
    g_launches += 2;
    STEPS_CUDA(cudaGetLastError());
    w.fuse_valid = false;
    if (g_fuse_eq12.load() != 0) {
        STEPS_CUDA(cudaMemsetAsync(fused_bits, 0xff, sizeof(unsigned long long), st));      // any bit pattern >= +inf: no limit yet
        t_fuse = Eq12Fuse{pos, soft, state5, std::fabs(G), B, eps, fused_bits};
    }
    rc = forces_impl(pos, mass, soft, N, 0, N, acc, mixed, stream);
    const bool was_on = t_fuse.out_bits != nullptr;
    t_fuse = NO_FUSE;
    if (rc != STEPS_OK) return rc;
    if (was_on) {
        w.fuse_token = FuseToken{pos, acc, soft, state5, N, std::fabs(G), B, eps, g_launches.load()};
        w.fuse_valid = true;
    }
    return STEPS_OK;
}

int steps_kick_close_adaptive(double* pos, double* vel, const double* acc, long long N, double* state5, double B,
                              steps_stream_t stream)
{
    if (!pos || !vel || !acc || !state5 || N < 1) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, 1, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = claim_scratch(g_ws[dev], st);
    if (rc != STEPS_OK) return rc;
    double* coef6 = g_ws[dev].mom_partial + 2 * MOM_BLOCKS;
    close_coefficients_kernel<<<1, 32, 0, st>>>(reinterpret_cast<RunState*>(state5), B, coef6);
    const long long M = 3 * N;
    long long blocks = (M + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    kick_drift_dev_kernel<<<(int)blocks, 256, 0, st>>>(pos, vel, acc, M, coef6);
    g_launches += 2;
    STEPS_CUDA(cudaGetLastError());
    return release_scratch(g_ws[dev], st);
}

double steps_hubble(double a, const steps_cosmology* c)
{
    return c->H0 * std::sqrt(c->Omega_m / (a * a * a) + c->Omega_r / (a * a * a * a) + c->Omega_L +
                             c->Omega_k / (a * a));
}

double steps_scale_factor_rk4(double a, double dt, const steps_cosmology* c)
{
    auto f = [c](double s) { return s * steps_hubble(s, c); };
    const double k1 = f(a), k2 = f(a + 0.5 * dt * k1), k3 = f(a + 0.5 * dt * k2), k4 = f(a + dt * k3);
    return a + dt / 6.0 * (k1 + 2.0 * (k2 + k3) + k4);
}

int steps_kdk_schedule(double a_n, double dt, double G, const steps_cosmology* c, double* out6)
{
    if (!c || !out6 || !(a_n > 0.0)) return STEPS_EINVAL;
    const bool is_static = (c->H0 == 0.0);
    const double H_n = is_static ? 0.0 : steps_hubble(a_n, c);
    const double a_1 = is_static ? a_n : steps_scale_factor_rk4(a_n, dt, c);
    const double H_1 = is_static ? 0.0 : steps_hubble(a_1, c);
    out6[0] = 1.0 - H_n * dt;
    out6[1] = 0.5 * dt * G / (a_n * a_n * a_n);
    out6[2] = dt;
    out6[3] = 1.0 / (1.0 + H_1 * dt);
    out6[4] = 0.5 * dt * G / (a_1 * a_1 * a_1) * out6[3];
    out6[5] = a_1;
    return STEPS_OK;
}

int steps_momentum(const double* vec, const double* mass, long long N, double* out4, steps_stream_t stream)
{
    if (!vec || !mass || !out4 || N < 1) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, 1, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = claim_scratch(g_ws[dev], st);
    if (rc != STEPS_OK) return rc;
    momentum_stage1<<<MOM_BLOCKS, 256, 0, st>>>(vec, mass, N, g_ws[dev].mom_partial);
    momentum_stage2<<<1, 32, 0, st>>>(g_ws[dev].mom_partial, MOM_BLOCKS, out4);
    g_launches += 2;
    STEPS_CUDA(cudaGetLastError());
    return release_scratch(g_ws[dev], st);
}

int steps_timestep(const double* pos, const double* acc, const double* soft, long long N, double coef, double B,
                   double eps, double dt_max, double* dt_out, steps_stream_t stream)
{
    if (!pos || !acc || !soft || !dt_out || N < 1) return STEPS_EINVAL;
    if (!(eps > 0.0) || !(dt_max > 0.0)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, 1, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = claim_scratch(g_ws[dev], st);
    if (rc != STEPS_OK) return rc;
    timestep_stage1<<<MOM_BLOCKS, 256, 0, st>>>(pos, acc, soft, N, coef, B, eps, dt_max, g_ws[dev].mom_partial);
    timestep_stage2<<<1, 32, 0, st>>>(g_ws[dev].mom_partial, MOM_BLOCKS, dt_out);
    g_launches += 2;
    STEPS_CUDA(cudaGetLastError());
    return release_scratch(g_ws[dev], st);
}

double steps_timestep_coefficient(double G, double a) { return std::fabs(G) / (a * a * a); }

int steps_force_residual(const double* pos, const double* acc, long long N, double B, double* out2, steps_stream_t stream)
{
    if (!pos || !acc || !out2 || N < 1) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    rc = ensure_workspace(dev, 1, reinterpret_cast<cudaStream_t>(stream));
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = claim_scratch(g_ws[dev], st);
    if (rc != STEPS_OK) return rc;
    residual_stage1<<<MOM_BLOCKS, 256, 0, st>>>(pos, acc, N, B, g_ws[dev].mom_partial);
    residual_stage2<<<1, 32, 0, st>>>(g_ws[dev].mom_partial, MOM_BLOCKS, out2);
    g_launches += 2;
    STEPS_CUDA(cudaGetLastError());
    return release_scratch(g_ws[dev], st);
}

int steps_sort_radial(const double* pos, long long N, long long* perm, steps_stream_t stream)
{
    if (!pos || !perm || N < 1 || N > (1ll << 31) - IB) return STEPS_EINVAL;
    if (misaligned(pos) || misaligned(perm)) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = ensure_workspace(dev, 1, st);
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    size_t temp_bytes = 0;
    STEPS_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, temp_bytes, (const double*)nullptr, (double*)nullptr, (const long long*)nullptr,
                                               (long long*)nullptr, (int)N, 0, 64, st));
    const size_t arr = (sizeof(double) * (size_t)N + 255) / 256 * 256;
    const size_t need = 3 * arr + temp_bytes;
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (need > w.sort_bytes) {
            if (stream_is_capturing(st)) return STEPS_ECAPTURE;
            STEPS_CUDA(cudaDeviceSynchronize());
            cudaFree(w.sort_buf); w.sort_buf = nullptr; w.sort_bytes = 0;
            if (cudaMalloc(&w.sort_buf, need) != cudaSuccess) { cudaGetLastError(); return STEPS_ENOMEM; }
            w.sort_bytes = need;
        }
    }
    rc = claim_scratch(w, st);
    if (rc != STEPS_OK) return rc;
    unsigned char* base = static_cast<unsigned char*>(w.sort_buf);
    double* keys_in = reinterpret_cast<double*>(base);
    double* keys_out = reinterpret_cast<double*>(base + arr);
    long long* idx_in = reinterpret_cast<long long*>(base + 2 * arr);
    radial_keys_kernel<<<(int)((N + 255) / 256), 256, 0, st>>>(pos, N, keys_in, idx_in);
    STEPS_CUDA(cub::DeviceRadixSort::SortPairs(base + 3 * arr, temp_bytes, keys_in, keys_out, idx_in, perm, (int)N, 0, 64, st));
    g_launches += 1;
    STEPS_CUDA(cudaGetLastError());
    return release_scratch(w, st);
}

int steps_permute(const double* src, long long N, int ncomp, const long long* perm, double* dst, steps_stream_t stream)
{
    if (!src || !perm || !dst || N < 1 || ncomp < 1 || src == dst) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    permute_kernel<<<(int)((N + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(src, N, ncomp, perm, dst);
    g_launches++;
    STEPS_CUDA(cudaGetLastError());
    return STEPS_OK;
}

int steps_near_fraction(const double* pos, const double* mass, const double* soft, long long N, double* out2, steps_stream_t stream)
{
    if (!pos || !mass || !soft || !out2 || N < 1 || N > (1ll << 31) - IB) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    rc = ensure_workspace(dev, N, st);
    if (rc != STEPS_OK) return rc;
    Workspace& w = g_ws[dev];
    rc = claim_scratch(w, st);
    if (rc != STEPS_OK) return rc;
    const int nt = (int)ntiles_of(N);
    TileF64* tiles = reinterpret_cast<TileF64*>(w.tiles);
    unsigned long long* counts = reinterpret_cast<unsigned long long*>(w.mom_partial);
    STEPS_CUDA(cudaMemsetAsync(counts, 0, 2 * sizeof(unsigned long long), st));
    prep_tiles<TileF64><<<nt, TJ, 0, st>>>(pos, mass, soft, N, tiles, nullptr);
    near_pairs_kernel<TileF64><<<(int)((N + WARP_I - 1) / WARP_I), 128, 0, st>>>(pos, soft, N, tiles, nt, counts);
    counts_to_double_kernel<<<1, 32, 0, st>>>(counts, out2);
    g_launches += 3;
    STEPS_CUDA(cudaGetLastError());
    return release_scratch(w, st);
}

int steps_reserve(long long N)
{
    if (N < 1) return STEPS_EINVAL;
    int dev;
    int rc = current_device(&dev);
    if (rc != STEPS_OK) return rc;
    return ensure_workspace(dev, N, nullptr);
}

void steps_shutdown(void)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    int cur = 0;
    cudaGetDevice(&cur);
    for (int d = 0; d < MAX_DEVICES; ++d) {
        Workspace& w = g_ws[d];
        if (!w.tiles && !w.mom_partial && !w.h_pos) continue;
        cudaSetDevice(d);
        cudaDeviceSynchronize();
        cudaFree(w.tiles); cudaFree(w.partials); cudaFree(w.plan); cudaFree(w.gm); cudaFree(w.acc_dd); cudaFree(w.sym_records);
        cudaFree(w.mom_partial); cudaFree(w.sort_buf);
        cudaFree(w.h_pos); cudaFree(w.h_mass); cudaFree(w.h_soft); cudaFree(w.h_acc);
        if (w.ev0) { cudaEventDestroy(w.ev0); cudaEventDestroy(w.ev1); }
        if (w.scratch_done) cudaEventDestroy(w.scratch_done);
        w = Workspace();
    }
    cudaSetDevice(cur);
}

long long steps_workspace_bytes(long long N)
{
    if (N < 1) return 0;
    size_t bytes = tile_bytes_max() * (size_t)ntiles_padded(N) + partial_bytes(N) + sizeof(double) * MOM_BLOCKS * 4 +
                   sym_plan_bytes(nblocks_of(N)) +
                   sizeof(GroupMeta) * (size_t)nblocks_of(N) * (IB / SPLITJ_GROUP);
    if (sym_eligible(N)) bytes += sizeof(double) * 6 * (size_t)N + sym_record_bytes(sym_panel_items_for(N));
    return (long long)bytes;
}

const char* steps_strerror(int code)
{
    switch (code) {
        case STEPS_OK: return "ok";
        case STEPS_EINVAL: return "invalid argument (null or misaligned pointer, N < 1, or bad range)";
        case STEPS_ECUDA: return "CUDA runtime error (see steps_last_cuda_error)";
        case STEPS_EUNSUPPORTED: return "device is not compute capability 10.x (sm_100a build, no fallback)";
        case STEPS_ENOMEM: return "workspace allocation failed";
        case STEPS_ECAPTURE: return "workspace must be allocated (steps_reserve) before the stream is captured into a CUDA graph";
        case STEPS_ETOOLARGE: return "steps_forces_static: N exceeds STEPS_STATIC_MAX_N = 16384 (fixed scratch array); use steps_reserve + steps_forces";
        default: return "unknown error code";
    }
}

int steps_last_cuda_error(void) { return g_last_cuda_error; }
int steps_version(void) { return 100; }
long long steps_kernel_launch_count(void) { return g_launches.load(); }

int steps_set_option(const char* key, long long value)
{
    if (!key) return STEPS_EINVAL;
    if (std::strcmp(key, "driver") == 0) { g_driver = (int)value; return STEPS_OK; }
    if (std::strcmp(key, "profile") == 0) { g_profile = (int)value; return STEPS_OK; }
    if (std::strcmp(key, "sym") == 0) { g_sym_enabled = (int)value; return STEPS_OK; }
    if (std::strcmp(key, "splitj") == 0) { g_splitj = (int)value; return STEPS_OK; }
    if (std::strcmp(key, "box_gsplit") == 0) { g_box_gsplit = (int)value; return STEPS_OK; }
    if (std::strcmp(key, "fuse_eq12") == 0) { g_fuse_eq12 = (int)value; return STEPS_OK; }
    if (std::strcmp(key, "sym_panel_items") == 0) {
        if (value < 1) return STEPS_EINVAL;
        g_sym_panel_items = value;
        return STEPS_OK;
    }
    return STEPS_EINVAL;
}

double steps_last_force_kernel_ms(void)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return -1.0;
    Workspace& w = g_ws[dev];
    if (!w.ev_valid) return -1.0;
    float ms = 0.0f;
    if (cudaEventSynchronize(w.ev1) != cudaSuccess || cudaEventElapsedTime(&ms, w.ev0, w.ev1) != cudaSuccess) return -1.0;
    return (double)ms;
}

int steps_pair_symmetric(long long N, int mixed) { return N >= 1 && sym_eligible(N, mixed != 0) && g_driver.load() == 0 ? 1 : 0; }

int steps_persistent_grid(int mixed)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return 0;
    return mixed ? g_ws[dev].grid_mixed : g_ws[dev].grid_fp64;
}

}  // extern "C"
