/*
 * enuf.h -- C ABI of the B200-native ENUF reciprocal-space library (libenuf_b200.so).
 *
 * ENUF = Ewald summation based on the non-uniform FFT (arxiv 2004.12484).  Citations
 * are PAPER.md:<line> of the paper text; R-numbers are the readings listed in DESIGN.md.
 *
 * What one evaluation computes (section II.C, and :487-507, section III.A):
 *   a1  wrap x = r/L (:301), bin particles by grid tile (counting sort)
 *   a2  spreading  g[l] = sum_j q_j phi(u_jx-l_x) phi(u_jy-l_y) phi(u_jz-l_z)      (:491)
 *   a3  forward 3D FFT of g on the oversampled n^3 grid, n = sigma*M              (:491)
 *   a4  scaling: S~(n) = g^[n]/D(n) for 0<|n|<=k_cut; E = (1/(2 pi L)) sum f^2 w |S~|^2
 *       with w(n) = exp(-(pi n)^2/(alpha L)^2)/n^2 (Eq. 38, :310); subdividing (:493)
 *   a5  inverse 3D FFT of the scaled spectrum (one field, or three for the ik variant)
 *   a6  interpolating back onto the particles as forces (Eq. 41-42, :332-340)
 *   a7  energy reduction to one fp64 scalar
 * Units: 1/(4 pi eps0) = 1 and eps_r = 1 (R1).  E is the reciprocal-space energy only
 * (includes i = j terms, no self / real-space / background term, R12-R13).
 *
 * Conventions for every entry point
 *   - returns ENUF_OK (0) or a negative enuf_status; enuf_last_error() then holds a
 *     thread-local message (for ENUF_ECUDA the CUDA error string).  No exception and no
 *     CPU fallback: without a CUDA device every compute call fails with ENUF_ECUDA.
 *   - "device pointer" = CUDA device memory of the plan's precision (float or double);
 *     "host pointer" = ordinary (preferably pinned) host memory.
 *   - the plan owns all workspace; nothing is allocated inside an evaluation.
 *   - a plan is not thread-safe; different plans may be used from different threads.
 */
#ifndef ENUF_H
#define ENUF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct enuf_plan enuf_plan; /* opaque */

enum enuf_status {
    ENUF_OK = 0,
    ENUF_EINVAL = -1, /* bad argument (message says which)            */
    ENUF_ENOMEM = -2, /* host or device allocation failed              */
    ENUF_ECUDA = -3,  /* a CUDA runtime call or kernel launch failed   */
    ENUF_ESTATE = -4  /* call not allowed in the plan's current state  */
};

/* keys of enuf_plan_set(); values are passed as double */
enum enuf_option {
    ENUF_OPT_PRECISION = 1,      /* ENUF_F32 (default) | ENUF_F64; only before the first evaluation */
    ENUF_OPT_WINDOW = 2,         /* ENUF_WINDOW_KAISER_BESSEL (default) | ENUF_WINDOW_GAUSSIAN (R6) |
                                    ENUF_WINDOW_BSPLINE: centred cardinal B-spline of order 2m (:266) |
                                    ENUF_WINDOW_SINC_POWER: sinc(pi c d)^2m, c = (2 - 1/sigma)/(2m) (:266) */
    ENUF_OPT_FORCE_VARIANT = 3,  /* ENUF_FORCE_ANALYTIC (default) | ENUF_FORCE_IK (paper, Eq. 41)   */
    ENUF_OPT_SLATER_LAMBDA = 4,  /* decay length of the Slater density Eq. 51 (:407); 0 = point (R19) */
    ENUF_OPT_NUM_PARTICLES = 5,  /* lower N for the next calls, 0 <= N <= planned capacity          */
    ENUF_OPT_PROFILE = 6,        /* 1: record per-stage CUDA-event times (enuf_plan_stage_ms)        */
    ENUF_OPT_KEEP_SPECTRUM = 7,  /* 1: also store S~(n) so enuf_plan_structure_factor() can read it  */
    ENUF_OPT_SPREAD_ZCHUNK = 8,  /* tuning: the spreading CTAs take fixed pieces of that many grid planes of one
                                    column (integer, 1..n) instead of the default, equal shares of all
                                    (column, plane) slabs, one per resident CTA.  Pieces shorter than 2m planes
                                    make the rounding order of the shared planes run-dependent (R22)        */
    ENUF_OPT_PDL = 10,           /* 1 (default): the kernels of an evaluation are launched with programmatic
                                    dependent launch -- each may be scheduled while its predecessor still runs
                                    and waits for it on the device (griddepcontrol), which hides the launch
                                    latency between the 11 kernels; 0: plain stream order                  */
    ENUF_OPT_SPREAD_SPARSE = 11, /* tuning, fp32: -1 (default) the plan picks per evaluation, 1 / 0 force the
                                    spreading kernel's eight-stage ring of 32-particle rounds (made for < ~12
                                    staged particles per slab and column) on / off; results are the same   */
    ENUF_OPT_CUDA_GRAPH = 9      /* 1: the launches of one evaluation are captured into a CUDA graph
                                    the second time the same (r, q, F) pointers and N are passed, and
                                    replayed while they stay the same (an MD loop that updates r in
                                    place); any enuf_plan_set call drops the graph.  Ignored while
                                    ENUF_OPT_PROFILE is on.  For the launch-bound small systems.     */
};

enum { ENUF_F32 = 0, ENUF_F64 = 1 };
enum { ENUF_WINDOW_GAUSSIAN = 0, ENUF_WINDOW_KAISER_BESSEL = 1, ENUF_WINDOW_BSPLINE = 2, ENUF_WINDOW_SINC_POWER = 3 };
enum { ENUF_FORCE_ANALYTIC = 0, ENUF_FORCE_IK = 1 };

/* stage indices of enuf_plan_stage_ms() */
enum enuf_stage {
    ENUF_STAGE_BIN = 0,     /* a1: histogram (+ zeroing of the grid planes that two spreading pieces share), scan,
                               scatter, window rows of the sorted particles */
    ENUF_STAGE_SPREAD = 1,  /* a2: grid values are stored once; only the planes two pieces of a column share are reduced */
    ENUF_STAGE_FFT = 2,     /* a3 + a4 + a5 */
    ENUF_STAGE_GATHER = 3,  /* a6 */
    ENUF_STAGE_ENERGY = 4,  /* a7 */
    ENUF_NUM_STAGES = 5
};

/*
 * Create a plan (step a0: tables of the window transform Phi(k), the influence function
 * f^2 w(|n|^2), FFT twiddles, workspace).
 *   N      particle capacity, >= 0
 *   L      cubic box edge (> 0); positions are wrapped into [0, L) internally (R10)
 *   alpha  Ewald convergence parameter (> 0)
 *   k_cut  reciprocal cutoff n_c in integer wavevectors: modes 0 < |n|^2 <= k_cut^2 (R4);
 *          1 <= k_cut <= M/2 (R5)
 *   M      NFFT bandwidth per dimension (Eq. 33, :272), any integer >= 2 k_cut
 *   sigma  oversampling factor sigma_s > 1 (:348, :360); n = sigma*M (to 1e-9) must be 32, 64, 128 or 256 -- the fused,
 *          pruned FFT: sigma = 2 with M a power of two, or any other M with sigma = n/M (M = 170, n = 256: 1.506) --
 *          or 48, 96, 192, 384: sigma = 1.5 with M = 32 ... 256, on a plain (slower) FFT path
 *   m      window cut-off: stencil of 2m+1 grid points per dimension (:268, R8), 1 <= m <= 6
 * Defaults: fp32, Kaiser-Bessel window, analytic-derivative forces, point charges,
 * the legacy default stream.  *out is set to NULL on failure.
 */
int enuf_plan_create(enuf_plan **out, int64_t N, double L, double alpha, int k_cut, int M,
                     double sigma, int m);

/*
 * The same for an orthorhombic periodic box with edges Lb[0..2] = (Lx, Ly, Lz) (host pointer, copied).  The
 * paper treats the cubic box and names other boxes as motivation (:35, :609); this is the Ewald
 * sum of such a cell written the same way (reading R26): x_d = r_d / L_d, wave vectors
 * k = 2 pi h with h = (nx/Lx, ny/Ly, nz/Lz), V = Lx Ly Lz,
 *   E~    = (1/(2 pi V)) sum_K f^2 exp(-pi^2 |h|^2/alpha^2)/|h|^2 |S~(n)|^2,
 *   K     = { n != 0 : |h| Lmax <= k_cut }, Lmax = max(Lx, Ly, Lz)  (every |n_d| <= k_cut L_d/Lmax <= k_cut),
 * ONE grid size n = sigma*M in all three directions (grid spacing L_d/n), forces -(q n/(pi V L_d)) sum Psi phi' phi phi
 * (analytic) or (2 q/V) sum B_d phi phi phi with b^_d = -i h_d psi^ (ik).  Equal edges give enuf_plan_create
 * exactly.  Everything else (options, evaluation calls, sharded halves, layouts) is the same;
 * enuf_plan_structure_factor takes modes of this K; enuf_real_space returns ENUF_EINVAL (cubic only).
 */
int enuf_plan_create_box(enuf_plan **out, int64_t N, const double *Lb, double alpha, int k_cut, int M,
                         double sigma, int m);

/* Change an option (see enuf_option).  Tables are rebuilt lazily at the next evaluation. */
int enuf_plan_set(enuf_plan *plan, int key, double value);

/* CUDA stream all work of the plan is issued to (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream); NULL = legacy default stream. */
int enuf_plan_set_stream(enuf_plan *plan, void *cuda_stream);

/*
 * One evaluation of the whole path a1..a7.
 *   r  device pointer, N x 3 row-major (x, y, z per particle), any real value
 *   q  device pointer, N charges; particles with q == 0 get F = 0 and are skipped
 *   F  device pointer, N x 3, OVERWRITTEN (not accumulated), caller's particle order
 *   E  host pointer to one double, or NULL.  If non-NULL the plan's stream is
 *      synchronised and *E receives E_rec; if NULL the call is fully asynchronous and
 *      the energy can be fetched later with enuf_plan_energy().
 * Caller owns r, q, F; they must stay valid until the stream has finished the call.
 */
int enuf_energy_forces(enuf_plan *plan, const void *r, const void *q, void *F, double *E);

/* Same, with HOST buffers: copies r, q to plan-owned device staging, evaluates, copies F
 * back, synchronises.  E may be NULL.  (The end-to-end path bench.py times.)
 * q_host may be NULL: the charges of the previous host call on this plan stay resident on the
 * device and are reused (an MD loop moves positions, not charges); ENUF_ESTATE if there was no
 * previous host call, or the workspace was re-allocated since. */
int enuf_energy_forces_host(enuf_plan *plan, const void *r_host, const void *q_host,
                            void *F_host, double *E);

/*
 * Sharded evaluation over several GPUs (the paper's HP-ENUF, section III.B).
 * The structure factor is additive over arbitrary particle subsets (Eq. 61, :533-540): every
 * rank holds a plan with the SAME (L, alpha, k_cut, M, sigma, m, options) and its OWN particles,
 * and one evaluation is
 *
 *   enuf_spectrum_partial(plan, r, q, F)       a1, a2 and the X, Y forward FFT passes on the
 *                                              rank's particles (F of its q == 0 particles is
 *                                              zeroed here, so F is the same buffer as below)
 *   all-reduce (sum) over ranks of the buffer  enuf_plan_spectrum_buffer() returns: `count`
 *                                              reals of the plan's precision, the half spectrum
 *                                              [z][ky'][kx] (complex, kx < Kxp, ky' < 2 k_cut + 1)
 *                                              after the X and Y passes -- linear in the charges.
 *                                              The caller does it (ncclAllReduce / torch.distributed
 *                                              on the plan's stream): "sums S_i(n) ... broadcasts",
 *                                              PAPER.md:542.  With one rank it is skipped.
 *   enuf_forces_from_spectrum(plan, F, E)      a4 .. a7 on the summed buffer: Z pass with scaling
 *                                              and energy, inverse passes (replicated on every
 *                                              rank), gather onto the rank's own particles.
 *
 * E is the energy of the WHOLE system (identical on all ranks up to nothing: same input bytes,
 * same fixed-order reduction); F holds the forces on the rank's own particles from all
 * particles of all ranks.  No force exchange is needed.  The device pointer returned by
 * enuf_plan_spectrum_buffer stays valid (and the same) until an option that reallocates the
 * workspace changes or the plan is destroyed.  enuf_forces_from_spectrum returns ENUF_ESTATE
 * unless enuf_spectrum_partial ran directly before it on this plan.
 */
int enuf_spectrum_partial(enuf_plan *plan, const void *r, const void *q, void *F);
int enuf_plan_spectrum_buffer(enuf_plan *plan, void **dev_ptr, size_t *count);
int enuf_forces_from_spectrum(enuf_plan *plan, void *F, double *E);

/*
 * Real-space (short-range) part of the Ewald sum and the self term -- the other two terms of
 * Eq. 25, so that E_total = E_real + E_rec - E_self on the device:
 *   E_real = 1/2 sum'_{i,j} q_i q_j B_U(d) erfc(alpha d)/d    over minimum-image pairs with d <= r_cut
 *            (Eq. 16-17, :176-181)
 *   F_i    = q_i sum'_j q_j B_F(d) [erfc(alpha d)/d^2 + (2 alpha/sqrt(pi)) exp(-alpha^2 d^2)/d] (r_i-r_j)/d
 *            (Eq. 29, :243 -- printed without q_i, the unit vector and the 1/d of the Gaussian term;
 *            the bracket here is -d/dd [erfc(alpha d)/d], reading R24)
 *   E_self = (alpha/sqrt(pi)) sum_i q_i^2                      (Eq. 24, :216; SUBTRACTED in Eq. 25, R13)
 * B_U, B_F are the Slater factors of Eq. 57-58 (:434-436) with r/lambda, lambda = ENUF_OPT_SLATER_LAMBDA;
 * lambda = 0 (default): point charges, B_U = B_F = 1.  Particles are sorted into a linked-cell list
 * with cells smaller than the cutoff (the paper's "Near Distance" scheme, :511-515).
 *   r, q       device pointers as in enuf_energy_forces (plan's N, L, alpha, precision, stream)
 *   r_cut      real-space cutoff, 0 < r_cut <= L/2 (minimum image)
 *   accumulate 0: F is OVERWRITTEN with the real-space forces (F = 0 for q == 0 particles);
 *              1: they are ADDED to F (e.g. after enuf_energy_forces wrote the reciprocal part)
 *   F          device pointer N x 3, caller's particle order
 *   E_real, E_self  host pointers or NULL; if either is non-NULL the stream is synchronised.
 */
int enuf_real_space(enuf_plan *plan, const void *r, const void *q, double r_cut, int accumulate,
                    void *F, double *E_real, double *E_self);

/* Synchronise the plan's stream and return the energy of the last evaluation. */
int enuf_plan_energy(enuf_plan *plan, double *E);

/* Per-stage device times (milliseconds) of the last evaluation; needs ENUF_OPT_PROFILE.
 * Writes min(count, ENUF_NUM_STAGES) floats.  Synchronises the stream. */
int enuf_plan_stage_ms(enuf_plan *plan, float *ms, int count);

/* Mean per-stage device times over the evaluations made since ENUF_OPT_PROFILE was last
 * set (at most the last 128; each evaluation records its own CUDA events on the plan's
 * stream, so no synchronisation happens between evaluations).  *n_evals (may be NULL)
 * receives how many evaluations were averaged.  Synchronises the stream. */
int enuf_plan_stage_ms_mean(enuf_plan *plan, float *ms, int count, int *n_evals);

/* Number of kernel launches (this library's kernels, excluding memsets/copies) the last
 * evaluation issued. */
int enuf_plan_launch_count(const enuf_plan *plan);

/* Test / multi-GPU taps (valid after an evaluation; each synchronises the stream).
 *   enuf_plan_copy_field: the spread grid g (after a2) is NOT kept -- this returns the real-space
 *     field Psi (analytic variant) or B_x (ik) that the gather read, n^3 values [z][y][x],
 *     to a HOST buffer of the plan's precision.
 *   enuf_plan_structure_factor: S~(n) for `count` modes (nx, ny, nz triples, each within
 *     the cutoff sphere) into out[2*count] (re, im) as fp64; needs ENUF_OPT_KEEP_SPECTRUM. */
int enuf_plan_copy_field(enuf_plan *plan, void *host_out);
int enuf_plan_structure_factor(enuf_plan *plan, int64_t count, const int *modes, double *out);

/* Spread only (a1 + a2) into a HOST buffer n^3 [z][y][x] of the plan's precision.
 * Used by the grid-vs-grid parity tests. */
int enuf_spread_only(enuf_plan *plan, const void *r, const void *q, void *grid_host);

/* Bytes of device workspace the plan holds. */
size_t enuf_plan_workspace_bytes(const enuf_plan *plan);

void enuf_plan_destroy(enuf_plan *plan);

/* Thread-local message of the last failing call ("" if none). */
const char *enuf_last_error(void);

/*
 * Parameter rule, Eq. 31-32, host only:
 *   enuf_ncut            smallest integer n_c >= (alpha L/pi) sqrt(-ln delta)      (R14)
 *   enuf_alpha_from_rc   alpha with exp(-alpha^2 r_c^2) = delta                    (R15)
 *   enuf_rc_from_ncut    r_c = pi n_c / (alpha^2 L)                                (Eq. 32)
 * Return a negative value / NaN on bad arguments.
 */
int enuf_ncut(double alpha, double L, double delta);
double enuf_alpha_from_rc(double r_c, double delta);
double enuf_rc_from_ncut(int n_c, double alpha, double L);

/*
 * The parameter loop of the paper ("for a given accuracy delta and real-space cutoff r_c, alpha and
 * n_c follow from Eq. 31-32"; :254-262) as a plan constructor: alpha = sqrt(-ln delta) / r_c (R15),
 * k_cut = n_c = ceil((alpha L / pi) sqrt(-ln delta)) (R14), M = the smallest power of two >= 2 k_cut (R5; all five
 * BASELINE configs follow this rule), then enuf_plan_create(N, L, alpha, k_cut, M, sigma, m).
 * ENUF_EINVAL if delta is not in (0, 1), r_c <= 0, or sigma * M leaves {32, 64, 128, 256}.
 * enuf_plan_get reads back what was chosen: key = ENUF_GET_ALPHA / K_CUT / M / GRID (n = sigma M) / SUPPORT (m).
 */
enum { ENUF_GET_ALPHA = 1, ENUF_GET_K_CUT = 2, ENUF_GET_M = 3, ENUF_GET_GRID = 4, ENUF_GET_SUPPORT = 5 };
int enuf_plan_create_auto(enuf_plan **out, int64_t N, double L, double delta, double r_c, double sigma, int m);
int enuf_plan_get(const enuf_plan *plan, int key, double *value);

/*
 * Allocation-free entry point, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): the self term of the Ewald sum,
 *     *E_self = (alpha / sqrt(pi)) sum_i q_i^2            (Eq. 24; subtracted in Eq. 25, :223)
 * -- the value enuf_real_space returns as *E_self -- from N charges q (DEVICE pointer, fp32 or fp64 as `precision`
 * = ENUF_F32 / ENUF_F64 says) into E_self (DEVICE pointer to one double), on `cuda_stream` (NULL = legacy default
 * stream).  Asynchronous: the value is there when the stream reaches that point.  The sum is formed in fp64 in a
 * fixed order, so the result is reproducible bit by bit.  No plan is needed and nothing is allocated or freed: the
 * scratch of the reduction (per-CTA partial sums and a counter, 128.25 KiB) is a static device array inside the
 * library, held by every GPU that loads it until the process exits.  Hence:
 *   - N <= ENUF_SELF_STATIC_MAX_N (2^24); larger N returns ENUF_EINVAL and launches nothing (use enuf_real_space);
 *   - every call shares that array: calls that can overlap on the GPU (different streams, or several host threads)
 *     race with one another; successive calls on one stream are safe.
 * ENUF_EINVAL for a NULL E_self, NULL q with N > 0, N < 0, a bad precision or alpha; ENUF_ECUDA for CUDA errors.
 */
#define ENUF_SELF_STATIC_MAX_N 16777216
int enuf_self_energy_static(const void *q, int64_t N, int precision, double alpha, void *cuda_stream,
                            double *E_self);

/*
 * Host only, no CUDA call: checks the work decomposition the spreading kernel would use (step a2)
 * on a grid of n points (a multiple of 16; columns of 32 x 16 cells for n >= 128, 16 x 16 below), window cut-off m
 * (trimmed != 0: the 2m-plane stencils of fp32 Kaiser-Bessel, m >= 5), precision ENUF_F32 / ENUF_F64, a device of
 * num_sms multiprocessors, and zchunk as ENUF_OPT_SPREAD_ZCHUNK (0 = the default, equal shares): every (column,
 * plane) slab must lie in exactly one piece, no piece may be shorter than the planes it shares with its neighbour
 * (zchunk = 0), and every piece start must be among the starts whose shared planes are zeroed.  ENUF_OK, or
 * ENUF_EINVAL with the first violation in enuf_last_error.  *G_out: CTAs; *min / *max_slabs_out: slabs of the
 * least and the most loaded CTA (any of the three may be NULL).  A test tap.
 */
int enuf_spread_split_check(int n, int m, int precision, int trimmed, int num_sms, int zchunk, int *G_out,
                            int *min_slabs_out, int *max_slabs_out);

#ifdef __cplusplus
}
#endif
#endif /* ENUF_H */
