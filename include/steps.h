/*
 * steps.h -- C ABI of steps-b200: the data-parallel hot path of StePS (arXiv:1811.05903)
 * on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (citations: PAPER.md line numbers / equation numbers;
 * "reading #k": DESIGN.md section "Readings of the paper"):
 *
 *   (1) the O(N^2) direct-summation force of Eq. 8 (L88), first term, with G = 1 and
 *       without the a(t)^-3 factor (both enter through the kick coefficients):
 *
 *           acc_i = sum_{j != i} m_j g(|x_j - x_i|, h_i + h_j) (x_j - x_i),   g = calF / r,
 *
 *       calF(r, h) the spline-softened 1/r^2 of Eq. 3-4 (L53-61), evaluated with the PAIR
 *       softening h_i + h_j (Eq. 2, Eq. 8; reading #3).  j = i is skipped and a
 *       coincident distinct pair (r = 0) contributes 0 (reading #4).  This is "the most
 *       time-consuming part" (L96, L131) and the only super-linear step.
 *   (2) the kick-drift-kick leapfrog of Eq. 9-11 (L98-109) applied to Eq. 8 in comoving
 *       coordinates, as one fused O(N) kernel driven by scalar coefficients the host
 *       derives from the Friedmann equation (Eq. 1, RK4 per L127), followed by the one
 *       force evaluation per step the paper asks for (L96).
 *
 * Conventions common to every call
 *   - All array arguments are DEVICE pointers unless the name ends in _host.  The caller
 *     owns every buffer; the library keeps no pointer after the call returns.
 *   - Layout: pos, vel, acc are SoA, 3N contiguous doubles [x_0..x_{N-1} | y_0.. | z_0..];
 *     mass and soft are N doubles.  Pointers must be 16-byte aligned.  soft[i] is the
 *     paper's h_i (Eq. 7, support radius of the spline), NOT a Plummer epsilon.
 *   - Calls are stream-ordered on `stream` (a cudaStream_t; NULL = legacy default stream)
 *     and never synchronise the host, except that the FIRST call for a larger N than any
 *     seen before on this device (re)allocates the internal workspace (cudaDeviceSynchronize +
 *     cudaMalloc).  steps_reserve(N) does that allocation up front; steps_shutdown() frees it.
 *   - The workspace (tile records, partial records, reduction scratch) is ONE per device.  Calls
 *     on different streams of one device are therefore SERIALISED, not concurrent: a call on
 *     another stream than the previous one first waits on the device (cudaStreamWaitEvent) for
 *     the previous call's last kernel.  Host threads may call concurrently (internal mutex).
 *   - CUDA graphs: every call can be captured provided the workspace exists already; a call that
 *     would have to allocate while `stream` is being captured returns STEPS_ECAPTURE and launches
 *     nothing.  The cross-stream serialisation above does not reach into a capture: use one
 *     capturing stream per device at a time.
 *   - Results do not depend on particle order beyond rounding.  Radially sorted input
 *     (|x| ascending) is the fast path: the kernels classify (i-group, j-tile) pairs by
 *     their radial intervals into "far" (no pair can have r < h_i + h_j; branch-free
 *     Newtonian body) and "near" (full per-pair spline test).  Unsorted input only makes
 *     more tiles "near" -- slower, never wrong.
 *   - Return value: STEPS_OK (0) or a negative error code; steps_strerror() gives text.
 *     Nothing throws or aborts.  N = 1 is valid (acc = 0).  Non-finite inputs give
 *     non-finite outputs, not an error.  Numerical domain of the fast (far) bodies:
 *     pair separations must satisfy 2^-63 < r < 2^63 (r^2 is seeded through fp32), and the
 *     mixed path, which works on r / sqrt(m_j) in fp32, needs 1e-12 < r / sqrt(m_j) < 1e18
 *     for every far pair (sources that cannot guarantee it from their own softening and
 *     coordinates are routed through the slower exact body).
 *   - The device must be compute capability 10.x (sm_100a cubin only; no PTX fallback,
 *     no CPU fallback): otherwise STEPS_EUNSUPPORTED.
 */
#ifndef STEPS_B200_STEPS_H
#define STEPS_B200_STEPS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct CUstream_st *steps_stream_t; /* cudaStream_t */

enum {
    STEPS_OK = 0,
    STEPS_EINVAL = -1,       /* null pointer, N < 1, misaligned pointer, bad range */
    STEPS_ECUDA = -2,        /* CUDA runtime / launch error (steps_last_cuda_error() has the code) */
    STEPS_EUNSUPPORTED = -3, /* current device is not sm_100 */
    STEPS_ENOMEM = -4,       /* workspace allocation failed */
    STEPS_ECAPTURE = -5,     /* the call would have to allocate workspace while its stream is being captured into a CUDA
                                graph: call steps_reserve(N) (and, for steps_forces_periodic, one un-captured call) first */
    STEPS_ETOOLARGE = -6     /* steps_forces_static: N > STEPS_STATIC_MAX_N (its scratch is a fixed array) */
};

/* ---- force evaluation --------------------------------- */

/* fp64 path: every pair in fp64 (the reciprocal square root is seeded by the fp32 SFU and
 * refined in fp64).  Bar: max_i |acc_i - oracle_i| / |oracle_i| <= 1e-12.
 * Overwrites acc[0..3N).  pos/mass/soft are read only.
 * From N = 16,385 (9 blocks of 2,048 particles; mixed path: from 30,721, 16 blocks) the evaluation is PAIR-SYMMETRIC: every block pair whose radial
 * intervals are further apart than the largest pair softening is evaluated once and applied to both blocks (Newton's
 * third law; PAPER.md L131 counts the cost as N(N-1)/2 pair evaluations), the band of block pairs around the diagonal
 * goes through the one-sided kernel.  The split is decided on the device from the data; unsorted input, massless
 * particles or too few blocks fall back to the one-sided kernel for everything.  Results are bit-reproducible either way.
 * The symmetric part needs 48 B per particle + up to 1.5 GiB of partial records (steps_workspace_bytes). */
int steps_forces(const double *pos, const double *mass, const double *soft, long long N,
                 double *acc, steps_stream_t stream);

/* steps_forces (fp64 path, same operation, same bar, same argument meaning) for callers that cannot allocate device
 * memory: code under CUDA-graph capture, tight loops, harnesses that forbid cudaMalloc.  This call never calls cudaMalloc,
 * cudaFree or an allocating library routine, on the first call or any later one.  Its scratch (the tile records of
 * PAPER.md Eq. 3-4's sources and the split-j partial records) is a file-scope __device__ array of the library:
 * STEPS_STATIC_SCRATCH_BYTES (about 2.6 MiB) that every GPU which loads the library holds until the process exits.
 *   - N <= STEPS_STATIC_MAX_N = 16,384 (the range of the split-j driver, one 128-particle group per CTA); a larger N
 *     returns STEPS_ETOOLARGE and launches nothing.  Use steps_reserve + steps_forces there.
 *   - pos, mass, soft, acc: device pointers, caller-owned, as for steps_forces.  The result equals steps_forces' at the
 *     same N (same kernels, same launch shape).
 *   - Every call on a device shares the one array, which keeps the previous call's contents.  Nothing in it has to start
 *     at zero: each call rewrites every record it later reads.  Calls that OVERLAP on the GPU (two streams, two host
 *     threads, a captured graph replayed next to a live call) race on it: give them one stream or order them with events. */
#define STEPS_STATIC_MAX_N 16384
#define STEPS_STATIC_SCRATCH_BYTES 2755584
int steps_forces_static(const double *pos, const double *mass, const double *soft, long long N,
                        double *acc, steps_stream_t stream);

/* mixed path: pair arithmetic in fp32 (the paper's GPU runs were single precision, L159),
 * per-tile fp32 partial sums flushed into fp64 accumulators.
 * Bar: RMS relative error <= 2e-6, max <= 1e-4. */
int steps_forces_mixed(const double *pos, const double *mass, const double *soft, long long N,
                       double *acc, steps_stream_t stream);

/* The paper's multi-node decomposition (L139: node k computes floor(N/N_node) force
 * vectors against all particles): forces on particles i in [i_begin, i_end) only, against
 * all N sources.  acc_out is SoA over the range: 3*(i_end-i_begin) doubles
 * [ax | ay | az].  mixed != 0 selects the mixed path. */
int steps_forces_range(const double *pos, const double *mass, const double *soft, long long N,
                       long long i_begin, long long i_end, double *acc_out, int mixed,
                       steps_stream_t stream);

/* The same decomposition dealt ROUND-ROBIN ("deal the radially sorted order round-robin by tile so every
 * GPU gets the same far/near mix"): forces on the particles of the blocks first_block, first_block + block_stride, ...
 * (blocks of steps_block_size() = 2,048 consecutive particles; rank r of P passes first_block = r, block_stride = P)
 * against all N sources.  acc_out is SoA over the owned particles in ascending order, packed: 3 * cnt doubles with
 * cnt = the number of owned particles (every owned block is full except possibly the last block of the set).
 * STEPS_EINVAL for first_block outside the blocks of N or block_stride < 1. */
int steps_forces_blocks(const double *pos, const double *mass, const double *soft, long long N,
                        long long first_block, long long block_stride, double *acc_out, int mixed,
                        steps_stream_t stream);

/* The force evaluation shared among `world` ranks by WORK instead of by particles (PAPER.md L135-139 partitions the force
 * vectors; L131 counts the work as N(N-1)/2 pair evaluations -- this call partitions those): acc_part (3N doubles, SoA over
 * ALL particles) receives the contribution of the rank-th of `world` equal parts of the pair evaluations of steps_forces /
 * steps_forces_mixed -- of the band's tile visits and of the pair-symmetric block-pair items, each applied to both of its
 * blocks -- so that the SUM over the ranks of acc_part is the full result to rounding (each part is rounded to fp64 once).
 * Every rank holds all particles; the one exchange per step is a sum-reduction of 3N doubles (NCCL all-reduce, 25 MB at
 * N = 1M) instead of the all-gather of positions, and every rank then advances ALL particles (O(N), bit-identical on every
 * rank).  Each rank runs the pair-symmetric kernels at their single-GPU rate (steps_forces_blocks is one-sided).  Below the
 * pair-symmetric size (N < 16,385 fp64 / 30,721 mixed: under half a millisecond of work) rank 0 evaluates everything and the
 * other ranks return zeros.  STEPS_EINVAL for rank outside [0, world). */
int steps_forces_share(const double *pos, const double *mass, const double *soft, long long N, int rank,
                       int world, double *acc_part, int mixed, steps_stream_t stream);
int steps_block_size(void);

/* End-to-end convenience with HOST buffers (pageable or pinned): copies pos/mass/soft to
 * the device, evaluates the forces, copies acc back and synchronises `stream` before
 * returning.  Used by bench.py's e2e figure. */
int steps_forces_host(const double *pos_host, const double *mass_host, const double *soft_host,
                      long long N, double *acc_host, int mixed, steps_stream_t stream);

/* ---- radial order --------------------------------------------- */

/* perm (device, N int64, 16-byte aligned) = the particle indices in order of ascending |x| (keys |x|^2 in fp64; equal
 * keys keep their input order).  The force calls are correct for ANY particle order; radially ordered input is what
 * makes almost every (i-group, j-tile) pair "far" and keeps the pair-symmetric band narrow, so a long run re-sorts when
 * steps_near_fraction has grown.  Stream-ordered; allocates its buffers on first use for a larger N (cudaMalloc). */
int steps_sort_radial(const double *pos, long long N, long long *perm, steps_stream_t stream);
/* dst[c][k] = src[c][perm[k]] for the ncomp components of an SoA array (ncomp = 3 for pos/vel/acc, 1 for mass/soft);
 * src and dst must not overlap. */
int steps_permute(const double *src, long long N, int ncomp, const long long *perm, double *dst,
                  steps_stream_t stream);
/* Tile-classification statistics for the given order: out2 (device, 2 doubles) = {number of (128-particle i-group,
 * 256-source tile) pairs that are NOT far, number of all such pairs}. */
int steps_near_fraction(const double *pos, const double *mass, const double *soft, long long N, double *out2,
                        steps_stream_t stream);

/* ---- time integration ---------------------------------- */

/* Coefficients of one fused kick/drift pass.  With g_i = acc_i + B x_i the pass does
 *     v <- alpha_close v + beta_close g     (closing half kick of the PREVIOUS step)
 *     v <- alpha_open  v + beta_open  g     (opening half kick of THIS step)
 *     x <- x + gamma v                      (drift)
 * For Eq. 8 with reading #6 (the background term carries a^-3) and reading #8 (drag
 * explicit in the opening, implicit in the closing half kick), a step a_n -> a_{n+1} of
 * length dt has
 *     alpha_open = 1 - H_n dt            beta_open  = G a_n^-3 dt/2         gamma = dt
 *     alpha_close = 1/(1 + H_{n+1} dt)   beta_close = G a_{n+1}^-3 (dt/2)/(1 + H_{n+1} dt)
 * and B = (4 pi/3) rho_bar (G = 1 units).  The identity kick is alpha = 1, beta = 0.
 * steps_kdk_schedule() fills these from the cosmology.  `mixed` selects the force path. */
typedef struct {
    double alpha_close, beta_close;
    double alpha_open, beta_open;
    double gamma;
    double B;
    int mixed;
} steps_kdk_coeffs;

/* The fused O(N) pass alone (Eq. 9-10): updates vel and pos in place from acc. */
int steps_kick_drift(double *pos, double *vel, const double *acc, long long N,
                     const steps_kdk_coeffs *c, steps_stream_t stream);

/* One integrator step: steps_kick_drift, then ONE force evaluation at the new positions
 * into acc (L96).  Driver pattern: steps_forces once; per step one steps_kdk_step whose
 * *_close are the previous step's closing coefficients (identity on the first step);
 * a final steps_kick_drift with gamma = 0 and an identity opening kick closes the run. */
int steps_kdk_step(double *pos, double *vel, double *acc, const double *mass, const double *soft,
                   long long N, const steps_kdk_coeffs *c, steps_stream_t stream);

/* Host-side scalars (no device work).  Friedmann equation, Eq. 1 (L37). */
typedef struct {
    double H0, Omega_m, Omega_r, Omega_L, Omega_k; /* present-day values, code units */
} steps_cosmology;

double steps_hubble(double a, const steps_cosmology *c);
/* a(t + dt) by classical RK4 on da/dt = a H(a) (L127). */
double steps_scale_factor_rk4(double a, double dt, const steps_cosmology *c);
/* Fills the opening half kick, drift and closing half kick of the step a_n -> a_{n+1}
 * (a_{n+1} by RK4, H0 = 0 means static Newtonian mode, L92) into
 * out[0..5] = {alpha_open, beta_open, gamma, alpha_close, beta_close, a_next}. */
int steps_kdk_schedule(double a_n, double dt, double G, const steps_cosmology *c, double *out6);

/* Diagnostics (row a7): out4 (device, 4 doubles) = {sum m v_x, sum m v_y, sum m v_z,
 * sum m |v|}.  Deterministic fixed-order reduction. */
int steps_momentum(const double *vec, const double *mass, long long N, double *out4,
                   steps_stream_t stream);

/* Quasi-periodic boundary conditions, Eq. 5 (L65-70, first part): "only the leading
 * term of the sum in Eq. 5 is kept for each pair of particles" -- every separation x_j - x_i is replaced by its image of
 * smallest length in a cubic box of side L (component-wise d - L rint(d / L), ties to even), otherwise exactly
 * steps_forces / steps_forces_mixed (mixed != 0): same layout, same pair law with pair softening soft_i + soft_j, G = 1,
 * acc overwritten.  Positions need not lie inside [0, L): the fp64 path wraps separations, valid for |x_j - x_i| < 2^51 L;
 * the mixed path casts positions to fp32 first, so it keeps its accuracy only for positions within a few L of the box
 * (|x| / L < 2^22 is the hard limit of its wrap).  Fast path: CELL-ORDERED input (e.g. Morton order of a grid, see
 * synth.morton_order) -- the periodic counterpart of the radial order: groups of consecutive particles whose bounding
 * boxes are compact and cannot hold a softened pair share one image decision -- a lattice shift per component, plus a
 * FOLD (d' = e - copysign(L/2, e), one addition and one bit operation) of the components whose separations straddle half
 * the box -- and run the open-boundary far body; from N = 16,385 (fp64) / 161,793 (mixed) such pairs of groups of two
 * different blocks of 2,048 particles are evaluated ONCE and applied to both groups (Newton III, as steps_forces does).
 * Unordered input, or particles given many periods apart, go through the general wrapped body with the per-pair softening
 * test -- slower, never wrong.  Ties (a separation component of exactly L/2, measure zero) may pick either image.  The
 * image sum of Eq. 5 with the 2.6 L cut is steps_forces_periodic below.  STEPS_EINVAL additionally for L <= 0. */
int steps_forces_quasi_periodic(const double *pos, const double *mass, const double *soft, long long N,
                                double L, double *acc, int mixed, steps_stream_t stream);

/* Periodic boundary conditions, Eq. 5 (L65-70, second part): the sum over the periodic
 * images x - nL of every separation with the paper's cut |x - nL| < 2.6 L (strict), each image through the pair law with
 * pair softening soft_i + soft_j; fp64 path only (the images of a homogeneous box cancel to a small remainder).  Layout,
 * G = 1 and error behaviour as steps_forces_quasi_periodic; the result does not depend on which representative modulo L
 * the positions are given in (|x_j - x_i| < 2^51 L).  Cost: 74 images per pair inside the cut on average; a pair on its
 * own needs 179 candidates (all n.n <= 12 around its leading image), a pair of 128-particle groups of cell-ordered input
 * whose bounding boxes are compact and cannot hold a softened pair is pruned to the ~90-110 candidates that come within
 * the cut for some pair of the two boxes, and from N = 16,385 such pairs of groups of two different blocks of 2,048
 * particles are evaluated ONCE for both groups (the image sum of a pair is antisymmetric).  A particle's OWN images (j = i, n != 0) are summed like any other pair's: the triplet set is symmetric under
 * n -> -n, so they cancel to rounding (the oracle skips j = i altogether).  Softening up to h_i + h_j <= L/2 takes the
 * fast route (only the nearest image can then be softened); larger softening is handled image by image. */
int steps_forces_periodic(const double *pos, const double *mass, const double *soft, long long N, double L,
                          double *acc, steps_stream_t stream);

/* Adaptive global time step, Eq. 12 (L113-116):
 *     dt = min[ dt_max, min_i sqrt(2 eta_i eps / |A_i|) ],  eta_i = 2.8 soft[i]  (L116, literal),
 * A_i = coef (acc_i + B pos_i) = the acceleration the kick applies, without the drag (coef = G a^-3, reading #6/#11);
 * |A_i| = 0 puts no limit.  pos, acc: SoA 3N device doubles; soft: N; dt_out: ONE device double (stream-ordered, the
 * host is not synchronised -- read it back when the next step's coefficients are needed).  Exact minimum, so the
 * result does not depend on the reduction order.  STEPS_EINVAL for null pointers, N < 1, eps <= 0 or dt_max <= 0. */
int steps_timestep(const double *pos, const double *acc, const double *soft, long long N, double coef,
                   double B, double eps, double dt_max, double *dt_out, steps_stream_t stream);
/* Host scalar: the `coef` of steps_timestep at scale factor a, |G| a^-3 (Eq. 8 L88 with reading #6; |G| because the
 * reversed gravity of glass generation, G < 0, changes the direction of A_i, not its size). */
double steps_timestep_coefficient(double G, double a);

/* Device-resident adaptive stepping (second half): one KDK step whose length is Eq. 12 and whose
 * coefficients (Eq. 1 / RK4 of L127 / readings #8-#9, the arithmetic of steps_kdk_schedule) are computed ON THE DEVICE,
 * so that a run needs no host round trip between steps and a sequence of these calls can be captured in a CUDA graph.
 * state5 (device, 5 doubles) = {a, dt of the last step, alpha_close, beta_close, steps taken}; initialise it to
 * {a_0, 0, 1, 0, 0}.  Per call: dt = Eq. 12 from (pos, acc, soft) with coef = |G| a^-3; closing kick of the previous
 * step + opening kick + drift; force evaluation at the new positions into acc; state advanced to a_{n+1}.  acc must hold
 * the forces at the current positions on entry (steps_forces before the first call).  steps_kick_close_adaptive applies
 * the pending closing half kick (end of a run, or before velocities are read) and resets it to the identity.
 * G < 0 = reversed gravity (glass generation).  cosmo is read on the host at call time.
 * Eq. 12's minimum is FUSED into the last kernel of the call's force evaluation (it writes every acc_i anyway) and used by
 * the next call when that call follows directly -- same pos/acc/soft/state5 pointers, N, |G|, B, eps and no other call of
 * this library in between; otherwise the next call forms the minimum with a separate O(N) pass (always on the first step).
 * Consequence for the caller: between two consecutive calls, change pos, acc, soft or state5 only through this library
 * (as the contract above already demands of acc), or switch the shortcut off with steps_set_option("fuse_eq12", 0).
 * Both ways give bit-identical steps. */
int steps_kdk_step_adaptive(double *pos, double *vel, double *acc, const double *mass, const double *soft,
                            long long N, double *state5, const steps_cosmology *cosmo, double G, double B,
                            double eps, double dt_max, int mixed, steps_stream_t stream);
int steps_kick_close_adaptive(double *pos, double *vel, const double *acc, long long N, double *state5,
                              double B, steps_stream_t stream);

/* Glass generation (section 3.1).  Reversed gravity needs no call of its
 * own: it is G < 0 in steps_kdk_schedule (both the pair sum and the background term change sign, the uniform sphere
 * stays static).  This is its convergence monitor, the net force per particle g_i = acc_i + B pos_i:
 *     out2 (device, 2 doubles) = { sum_i |g_i|^2, max_i |g_i| }.
 * pos, acc: SoA 3N device doubles.  Deterministic fixed-order reduction, stream-ordered. */
int steps_force_residual(const double *pos, const double *acc, long long N, double B, double *out2,
                         steps_stream_t stream);

/* ---- housekeeping ------------------------------------------------------------------ */

int steps_reserve(long long N);          /* allocate workspace for up to N particles now */
void steps_shutdown(void);               /* free all workspace on all devices */
long long steps_workspace_bytes(long long N); /* bytes steps_reserve(N) allocates */
const char *steps_strerror(int code);
int steps_last_cuda_error(void);         /* cudaError_t of the last STEPS_ECUDA on this thread */
int steps_version(void);                 /* major*10000 + minor*100 + patch */
/* Number of kernels this library has launched since load (for bench.py's gpu_launches). */
long long steps_kernel_launch_count(void);
/* Tuning / testing knobs.  "driver": 0 = default force driver (persistent, bulk-TMA), 1 = the
 * simple one-CTA-per-i-block driver kept as an in-library cross-check.  "profile": 1 = bracket
 * the force kernel(s) of every later call with CUDA events recorded on the call's stream.
 * "sym": 0 = never use the pair-symmetric evaluation (default 1).  "sym_panel_items": how many
 * block-pair items (96 KiB of partial records each) the symmetric evaluation keeps in flight
 * (default 16384 = 1.5 GiB; the items are run in panels of this size).  "splitj": 0 = never use the split-j driver.
 * "fuse_eq12": 0 = steps_kdk_step_adaptive always forms Eq. 12's minimum in its own pass.  "box_gsplit": CTAs that share
 * one group's possibly-softened units in the periodic pair-symmetric evaluation (default 8).  Unknown key: STEPS_EINVAL. */
int steps_set_option(const char *key, long long value);
/* With "profile" on: device time in ms of the most recent force kernel launched on the current
 * device (waits for it to finish); -1 if none was recorded.  For a pair-symmetric evaluation: from the
 * start of the band kernel to the end of the last panel's reduce (all force kernels of the evaluation). */
double steps_last_force_kernel_ms(void);
/* 1 if a full force evaluation of N particles on the given path is set up pair-symmetrically (see steps_forces: fp64 from
 * N = 16,385, mixed from N = 30,721, and the "sym" option on), else 0.  Host-side eligibility only: the device still routes
 * everything through the one-sided kernel when the data do not allow the split (unsorted input, massless particles). */
int steps_pair_symmetric(long long N, int mixed);
/* Grid (CTA count) of the persistent force kernel on the current device: SMs x resident CTAs;
 * 0 before the first call of that path. */
int steps_persistent_grid(int mixed);

#ifdef __cplusplus
}
#endif
#endif /* STEPS_B200_STEPS_H */
