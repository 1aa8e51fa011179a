/* se_mobility.h -- C ABI of the B200-native far-field mobility product of SEASD.
 *
 * One operation: the far-field grand-mobility product  M.[F,T,S] -> [U,Omega,E]  for N polydisperse
 * spheres in a cubic, triply periodic box, by the Ewald split of Wang & Brady, arXiv 1506.08481
 * ("PAPER.md"): a real-space pair sum with cutoff r_c over a cell list (Sec. 3.3, Eq. 22 with
 * the Faxen laws Eq. 13-15 and the multipole expansion Eq. 17) plus a Spectral-Ewald wave-space sum in
 * the hybrid size-effect variant (Sec. 3.1-3.2: Eq. 41-46, 48, 50-52), minus the wave-space self terms
 * (Eq. 37) plus the one-body Faxen terms (Eq. 13-15).
 *
 * Conventions: inputs are the moments the particles exert ON THE FLUID, (F,T,S) = -(F^H,T^H,S^H) of
 * Eq. 7-9; outputs are (U - U^inf, Omega - Omega^inf, -E^inf) of Eq. 11, so that the operator is the
 * symmetric positive definite grand mobility of PAPER.md L92.  S and E are symmetric and traceless and
 * are stored as 5 components (xx, xy, xz, yy, yz); zz = -(xx+yy).  Everything is IEEE double.
 *
 * Every entry point returns an se_status and never throws, aborts or prints.  The library has no CPU
 * fallback: without a CUDA device every compute call returns SE_ERR_CUDA.
 *
 * Threading/streams: a plan owns one workspace, so at most one apply per plan may be in flight;
 * different plans may be used concurrently on different streams.
 */
#ifndef SE_MOBILITY_H
#define SE_MOBILITY_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct se_plan se_plan;       /* opaque; created, owned and freed by the library */

typedef enum {
    SE_OK = 0,
    SE_ERR_INVALID_ARG = 1,           /* bad size/parameter or NULL pointer; nothing was launched    */
    SE_ERR_UNSUPPORTED = 2,           /* valid request this build does not implement (e.g. P > 24)   */
    SE_ERR_ALLOC = 3,                 /* host or device allocation failed                            */
    SE_ERR_CUDA = 4,                  /* CUDA runtime error (text in se_last_error)                  */
    SE_ERR_CUFFT = 5                  /* cuFFT error                                                 */
} se_status;

/* flags for se_plan_set_flags (staged parity and profiling; default 0 = the full product) */
#define SE_SKIP_REAL     0x1u         /* leave out the real-space pair sum (a2)                       */
#define SE_SKIP_WAVE     0x2u         /* leave out the Spectral-Ewald wave-space sum (a3-a7)          */
#define SE_SKIP_SELF     0x4u         /* do not subtract the wave-space self terms (Eq. 37)           */
#define SE_SKIP_ONEBODY  0x8u         /* do not add the one-body Faxen terms (Eq. 13-15)              */
#define SE_TIMING        0x10u        /* record CUDA events between stages (se_plan_get_timings)      */
#define SE_CUFFT3D       0x40u        /* a4/a6 by cuFFT's batched 3-D real transforms and a separate k-space kernel.
                                         Without this flag, power-of-two grids 32 <= M <= 512 take the faster default:
                                         own transform kernels on transposed half spectra [kz][x][y], the x transforms
                                         fused with the k-space scaling (no cuFFT).  Other M always use cuFFT.       */

/* stage indices of se_plan_get_timings */
enum {
    SE_STAGE_SORT = 0,                /* a1: wrap, counting sorts by real-space cell and grid tile, packing */
    SE_STAGE_REAL = 1,                /* a2: real-space pair sum                                      */
    SE_STAGE_SPREAD = 2,              /* a3: Gaussian spreading onto the grid                         */
    SE_STAGE_FFT_FWD = 3,             /* a4: forward FFTs (own z kernel + cuFFT 2-D, or cuFFT 3-D)    */
    SE_STAGE_KSPACE = 4,              /* a5: fused k-space scaling                                    */
    SE_STAGE_FFT_INV = 5,             /* a6: inverse FFTs (cuFFT 2-D + own z kernel, or cuFFT 3-D)    */
    SE_STAGE_GATHER = 6,              /* a7: Gaussian gather                                          */
    SE_STAGE_EPILOGUE = 7,            /* a8: self / one-body terms, sum, un-permute                   */
    SE_NUM_STAGES = 8
};

/* Create a plan.  Derives Delta = L/M, the Gaussian shape (Eq. 41, 46) with shape
 * parameter m = sqrt(pi P) (Eq. 79) unless changed by se_plan_set_shape, cell and tile grids, creates
 * the cuFFT plans and allocates every workspace on the CURRENT CUDA device.
 *   out     receives the plan (set to NULL on failure)
 *   N       number of particles, >= 1
 *   L       edge of the cubic periodic box [0,L)^3, > 0
 *   radii   HOST pointer, N entries, each > 0; copied                        (a_i)
 *   xi      Ewald splitting parameter, > 0 (Beenakker convention)
 *   r_c     real-space cutoff: pairs with minimum-image distance r < r_c;  0 < r_c <= L/2  (L330)
 *   M       grid points per axis, even, >= P
 *   P       support points of the Gaussian per axis, 2 <= P <= 24
 *   eta0    solvent viscosity, > 0
 * Errors: SE_ERR_INVALID_ARG for any violated bound or NULL; SE_ERR_UNSUPPORTED for P > 24;
 * SE_ERR_ALLOC / SE_ERR_CUDA / SE_ERR_CUFFT when resources cannot be had. */
se_status se_plan_create(se_plan **out, int64_t N, double L, const double *radii,
                         double xi, double r_c, int M, int P, double eta0);

/* Gaussian shape parameter m of Eq. 46 (h ~ exp(-m^2/2) at the edge of the support), m > 0. */
se_status se_plan_set_shape(se_plan *plan, double m);

/* Lees-Edwards strain (Sec. 3.1, Sec. 3.2 L300-302 with Eq. 48): the periodic lattice
 * becomes a1 = (L,0,0), a2 = (gamma L, L, 0), a3 = (0,0,L) -- simple shear, flow along x, gradient along y.  Positions stay
 * physical Cartesian coordinates (any real value; wrapped on the sheared lattice internally).  The grid lives in the
 * fractional coordinate t = A^{-1} r, in which the Gaussian of Eq. 41 is isotropic; the strain enters through the metric
 * B^T.B of its derivatives when spreading and gathering (Eq. 42, 45, 48), through k = B.q in the Green's function (Eq. 43),
 * through the sheared minimum image of the real-space sum, and in se_self_image_blocks.  gamma = 0 (default) is the cubic
 * box and takes exactly the original code paths.  Any finite gamma is accepted; gamma and gamma + 1 describe the same
 * lattice.  Drops the cached configuration.  Errors: SE_ERR_INVALID_ARG for a non-finite value. */
se_status se_plan_set_strain(se_plan *plan, double gamma);

/* Performance knob: number of segments the x-sweep of the spreading kernel is cut into (0 = the plan's own choice);
 * gather_segments is accepted and ignored (the gather kernel balances its own work over the SMs).
 * Results do not depend on it beyond summation order. */
se_status se_plan_set_tuning(se_plan *plan, int spread_segments, int gather_segments);

/* Further performance knobs, one integer each (results do not depend on them beyond summation order):
 *   SE_OPT_REAL_OVERLAP  where the real-space sum (a2), which is independent of the wave-space pipeline, runs:
 *                        0 = on the caller's stream before the spreading; 1 = on a plan-owned low-priority stream
 *                        beside the whole wave pipeline; 2 = on that stream, started after the spreading (beside the
 *                        HBM-bound transforms).  Joined before the epilogue in every case.
 *   SE_OPT_REAL_CTAS     CTAs of the real-space kernel when it runs beside the wave pipeline (0 = one per cell).  Default: a
 *                        persistent grid of one CTA per SM and per 256 cells to walk, at most three per SM.
 *   SE_OPT_XY_PATH       reserved (round 1's cuFFT 2-D path was removed when the own y / fused x kernels replaced it);
 *                        SE_ERR_INVALID_ARG.
 *   SE_OPT_YZ_FUSED      1 = the y and z transforms of a direction in ONE kernel (thread-block
 *                        clusters exchanging through distributed shared memory; default for M <= 128), 0 = separate
 *                        z and y kernels.
 *   SE_OPT_GRAPH         1 = far_mobility_apply / _compressible keep the whole product as a plan-owned CUDA graph: the
 *                        first call runs plainly, the second captures the sequence on the caller's stream, later calls
 *                        with the same pointers, stream, flags and options replay it in one launch (the data behind
 *                        the pointers may change freely).  Default: 1 for M <= 128, where launch latency dominates,
 *                        else 0.  Never used on the legacy default stream, inside a caller's own capture, with
 *                        SE_TIMING or se_plan_debug_stop.
 *   SE_OPT_PAIR_CACHE    1 (default) = se_plan_set_positions also does the neighbour search of the real-space sum and
 *                        stores, per pair r < r_c, the separation and the 17 radial scalars of the pair (160 bytes + 4);
 *                        products on the cached configuration (pos == NULL, also far_mobility_apply_batch) then only
 *                        stream that list.  Costs about 1.3 real-space sums once and 164 bytes per ordered pair
 *                        (c4: 0.66 GB); 0 = recompute the pairs in every product.  If the list cannot be allocated the
 *                        products silently recompute.
 *   SE_OPT_SIZE_VARIANT  how the particle-size terms of the Faxen laws and of the multipole expansion enter the wave-space sum
 *                        (Sec. 3.2); unlike the knobs above this one changes the DISCRETISATION, i.e. the result at
 *                        a given P (all three converge to the same sum, Fig. 2):
 *                        0 = hybrid (default; L324: derivatives of the Gaussian in the spreading, Laplacian in wave space,
 *                            3 grids to wave space and 6 back);
 *                        1 = real-space (L298-304: derivatives of the Gaussian on both sides; 3 grids to wave space, 3 back,
 *                            the gather takes the d^2-weighted sums; the cheapest product, the largest P for a given accuracy);
 *                        2 = wave-space (L306-322, Eq. 49-52: only the Gaussian is spread and gathered, F, a^2 F, T, S and
 *                            a^2 S on grids of their own, every derivative a wave-vector factor; 21 grids to wave space and
 *                            21 back in seven spreading passes and four gather batches through cuFFT's 3-D transforms; the
 *                            smallest P for a given accuracy, about 6 products' worth of transforms; extra workspace of 24
 *                            half spectra, allocated by the first such product; its stage timings put the seven passes
 *                            under "spread" and the four batches under "gather"; se_plan_debug_stop is not available).
 *                        Both alternatives cover the compressible entry point, cached positions, batches and the
 *                        sheared lattice (se_plan_set_strain; Fig. 2 shows them at gamma = 0.5 as well).
 *   SE_OPT_GRID_FP32     1 = single-precision mesh (Fig. 6: the paper's GPU code computes in single precision): the
 *                        spread grids are rounded to fp32, transformed, scaled and transformed back in fp32 (cuFFT's 3-D
 *                        R2C / C2R) and widened again for the gather; everything on the particle side (Gaussians, the
 *                        accumulation of the spreading and of the gather, the real-space sum, the epilogue) stays fp64.
 *                        Changes the RESULT: relative error about 3e-7 .. 3e-6 against the fp64 product (bound 1e-5 in the
 *                        tests), the error floor of Fig. 6a.  Hybrid and real-space size variants, cubic or sheared box,
 *                        compressible entry point included; with the wave-space variant the product returns
 *                        SE_ERR_UNSUPPORTED.  Extra workspace (7 fp32 grids, 11 fp32 half spectra, cuFFT plans) is
 *                        allocated by the first such product.  0 (default) = double precision throughout.
 * Errors: SE_ERR_INVALID_ARG for an unknown key or a value out of range. */
enum { SE_OPT_REAL_OVERLAP = 0, SE_OPT_REAL_CTAS = 1, SE_OPT_XY_PATH = 2, SE_OPT_YZ_FUSED = 3, SE_OPT_GRAPH = 4, SE_OPT_PAIR_CACHE = 5,
       SE_OPT_SIZE_VARIANT = 6, SE_OPT_GRID_FP32 = 7, SE_NUM_OPTS = 8 };
se_status se_plan_set_option(se_plan *plan, int key, int value);

/* Bitwise OR of the SE_* flags above. */
se_status se_plan_set_flags(se_plan *plan, unsigned flags);

/* Fix the particle configuration for the following products (the iterative solver applies the
 * operator many times per configuration).  Runs a1 once (wrap, counting sorts, per-particle
 * Gaussian tables and indices) on cuda_stream; afterwards far_mobility_apply / far_mobility_apply_compressible
 * may be called with pos == NULL and then only refresh the moments (F, T, S, s) of the packed records.
 *   pos    [N][3] DEVICE, as in far_mobility_apply; NULL forgets the cached configuration
 * The cache is dropped by se_plan_set_shape and by any apply that passes pos != NULL.  With a cached configuration
 * the summation order is fixed, so repeated products are bitwise reproducible.  With SE_OPT_PAIR_CACHE (default) the call
 * also builds the pair list of the real-space sum (the paper prebuilds its real-space matrix per configuration likewise,
 * PAPER.md L332) and synchronises cuda_stream once to size it. */
se_status se_plan_set_positions(se_plan *plan, const double *pos, void *cuda_stream);

/* The product.  All pointers are DEVICE pointers to arrays the caller owns:
 *   pos    [N][3] row-major particle centres, any real value (wrapped into the box internally);
 *          NULL = the configuration given to se_plan_set_positions
 *   F, T   [N][3] force and torque on the fluid
 *   S      [N][5] stresslet on the fluid, (xx,xy,xz,yy,yz)
 *   U, Omega [N][3], E [N][5]  outputs, OVERWRITTEN (never accumulated into)
 *   cuda_stream   a cudaStream_t (NULL = default stream); the work is enqueued and the call returns
 *                 without synchronising.  Inputs must stay valid until the stream reaches the end.
 * Errors: SE_ERR_INVALID_ARG for NULL pointers (pos == NULL without se_plan_set_positions included);
 * SE_ERR_CUDA / SE_ERR_CUFFT on launch failure. */
se_status far_mobility_apply(se_plan *plan, const double *pos, const double *F, const double *T,
                             const double *S, double *U, double *Omega, double *E, void *cuda_stream);

/* Several right-hand sides on ONE configuration: the iterative solver applies the operator tens to
 * hundreds of times per configuration with only (F,T,S) changing (nested GMRES; the paper prebuilds
 * its real-space matrix per time step for that reason, L332), and block methods apply it to several vectors at once.
 *   pos    [N][3] DEVICE or NULL (= the configuration of se_plan_set_positions); when given, a1 runs once and the
 *          configuration stays cached afterwards, exactly as after se_plan_set_positions
 *   nrhs   number of right-hand sides, >= 1
 *   F, T   [nrhs][N][3] DEVICE;  S  [nrhs][N][5] DEVICE            (right-hand side r starts at offset r N 3, r N 5)
 *   U, Omega [nrhs][N][3], E [nrhs][N][5] DEVICE outputs, OVERWRITTEN
 * Results equal nrhs calls of far_mobility_apply (same arithmetic per right-hand side).  What is shared: the sorts and
 * per-particle tables (once), and in the real-space sum (a2) the neighbour search and every pair's erfc/exp and radial
 * functions, evaluated once per pair for up to four right-hand sides per launch.  The wave-space pipeline (a3-a7) runs per
 * right-hand side.  Flags as for far_mobility_apply.  The first call with a larger nrhs allocates 2 nrhs N 12 doubles
 * (synchronising the stream).  Errors: SE_ERR_INVALID_ARG, SE_ERR_ALLOC, SE_ERR_CUDA, SE_ERR_CUFFT. */
se_status far_mobility_apply_batch(se_plan *plan, const double *pos, int nrhs, const double *F, const double *T,
                                   const double *S, double *U, double *Omega, double *E, void *cuda_stream);

/* Compressible-solvent extension (Sec. 2.3, Eq. 24-34).  As far_mobility_apply with
 *   s_in   [N] DEVICE pressure moments s_j (paper's Eq. 25-26 sign: s > 0 is a fluid source), or NULL for none.
 *          Adds the source field grad psi (Eq. 26, split after Eq. 33-34) to U and E: one more spread grid
 *          and forward FFT, an (i k/k^2) term in the k-space pass, two more couplings in the real-space sum.
 *   s_out  [N] DEVICE, OVERWRITTEN with the interaction part 4 pi a_i^3 p'(r_i) of the pressure Faxen law
 *          (Eq. 28-31: pressure from F and S of all particles), or NULL: one more spectrum, inverse FFT and
 *          plain Gaussian gather, two more couplings in the real-space sum.
 * With s_in == NULL the outputs U, Omega, E equal those of far_mobility_apply.  The first call that passes
 * s_in or s_out allocates the extra grids and cuFFT plans (synchronous; later calls only enqueue).
 * Errors: as far_mobility_apply, plus SE_ERR_ALLOC / SE_ERR_CUFFT from that allocation. */
se_status far_mobility_apply_compressible(se_plan *plan, const double *pos, const double *F,
                                          const double *T, const double *S, const double *s_in,
                                          double *U, double *Omega, double *E, double *s_out,
                                          void *cuda_stream);

/* Self-image Ewald blocks (Sec. 4.2: the block-diagonal approximation of the grand
 * mobility behind the far-field preconditioner -- "for each particle, the approximation only considers the interactions
 * with its periodic images", by direct Ewald summation).  Writes, for every particle i, the 11 x 11 matrix that maps
 * its own (F[3], T[3], S[5]) to its own (U[3], Omega[3], E[5]) when only the particle and its periodic images are there:
 * one-body terms (Eq. 13-15) - wave-space self terms (Eq. 37) + real-space image sum + wave-space sum of the self pair.
 *   out    DEVICE, [N][11][11] row-major (row = output component, column = input component, stored 5-component S and E),
 *          OVERWRITTEN
 * Depends on the radii, L and eta0 only (not on xi, r_c, M, P: the sums are direct and converged to round-off).
 * Cost O(N): the lattice sums are done for three reference radii (every entry is a quadratic in a_i^2 besides the one-body
 * term) and interpolated per particle.  Enqueues two kernels on cuda_stream; no synchronisation.
 * Errors: SE_ERR_INVALID_ARG for NULL; SE_ERR_ALLOC / SE_ERR_CUDA. */
se_status se_self_image_blocks(se_plan *plan, double *out, void *cuda_stream);

/* End-to-end convenience: the same product with HOST arrays (pinned or pageable).  Copies the inputs
 * to plan-owned device buffers, runs far_mobility_apply on cuda_stream, copies the outputs back and
 * synchronises the stream before returning. */
se_status far_mobility_apply_host(se_plan *plan, const double *pos, const double *F, const double *T,
                                  const double *S, double *U, double *Omega, double *E, void *cuda_stream);

/* The same without the final synchronisation: the three copies in, the product and the three copies out are enqueued on
 * cuda_stream and the call returns.  With PINNED host arrays nothing blocks, so a caller with independent products can keep two
 * in flight -- two plans on two streams -- and the copies of one overlap the kernels of the other (c4: 292 -> 325 products/s).
 * The copies are hidden completely (348 products/s against 351 with resident inputs) by a three-stream pipeline around
 * far_mobility_apply: uploads on one stream, the products on a second, downloads on a third, two sets of device buffers, one
 * event per set and stage (bench.py's "e2e" leg is that pipeline).
 * The host arrays must stay valid, and the outputs must not be read, until the stream is synchronised; one plan carries one
 * product at a time (its device buffers are reused by the next call on it).  Errors as far_mobility_apply. */
se_status far_mobility_apply_host_async(se_plan *plan, const double *pos, const double *F, const double *T,
                                  const double *S, double *U, double *Omega, double *E, void *cuda_stream);

/* Staged outputs for parity tests (valid after the stream of the last apply has been synchronised).
 * which = 0: the three spread grids H_x,H_y,H_z, [3][M][M][M];  which = 1: the six returned grids
 * u~ (3), w~ (3), [6][M][M][M];  which = 2: the scalar grid of the compressible extension, [M][M][M]
 * (the spread pressure moments after SE_STAGE_SPREAD, the returned pressure grid p~ after SE_STAGE_FFT_INV).  dst is a HOST pointer with room for the whole array.  The spread
 * grids share storage with the returned grids and are only available from an apply made with flag
 * SE_SKIP_WAVE cleared and read through which = 0 BEFORE a later apply; tests use se_plan_debug_stop. */
se_status se_plan_copy_grids(se_plan *plan, int which, double *dst);

/* Debug: stop the wave pipeline after stage `stage` (SE_STAGE_SPREAD .. SE_STAGE_GATHER), or -1 for
 * the normal full run.  Used with se_plan_copy_grids for per-stage parity. */
se_status se_plan_debug_stop(se_plan *plan, int stage);

/* CUDA-event times in milliseconds of the stages of the last apply made with SE_TIMING set;
 * synchronises on the last event.  ms has SE_NUM_STAGES entries. */
se_status se_plan_get_timings(se_plan *plan, double *ms);

/* Number of kernel launches (own kernels, cuFFT excluded) the last apply enqueued. */
int se_plan_last_launch_count(const se_plan *plan);

/* Device bytes held by the plan (grids, sorted copies, cell tables, cuFFT work areas). */
size_t se_plan_workspace_bytes(const se_plan *plan);

/* Derived constants, for tests: out[0..6] = Delta, eta_se, alpha, m, cells per axis of the real-space
 * cell grid (as double), number of sweep segments of the spreading and of the gather kernel (as double). */
se_status se_plan_get_constants(const se_plan *plan, double *out);

/* Measurement aid for the "alu" roofline of the real-space kernel: runs independent double-precision FMA
 * chains on every SM of the current device on cuda_stream (NULL = default), times them with CUDA events and
 * writes the sustained rate in TFLOP/s (2 flop per FMA) to *tflops.  Synchronises the stream.
 * Errors: SE_ERR_INVALID_ARG for NULL, SE_ERR_CUDA without a device. */
se_status se_measure_fp64_peak(double *tflops, void *cuda_stream);

/* Text of the last error on this plan ("" if none); owned by the plan. */
const char *se_last_error(const se_plan *plan);

/* Release everything.  NULL is allowed. */
se_status se_plan_destroy(se_plan *plan);

/* Library version string, e.g. "se_mobility 0.2 (sm_100a)". */
const char *se_version(void);

/* The real-space pair sum (a2; Sec. 3.3 with the pair couplings of Eq. 13-17 on Eq. 22's J_R) WITHOUT a plan and without
 * any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it):
 *     [U, Omega, E]_i = sum over j != i, minimum image, r_ij < r_c, of the real-space Ewald couplings with [F, T, S]_j,
 * i.e. exactly what far_mobility_apply returns with flags SE_SKIP_WAVE | SE_SKIP_SELF | SE_SKIP_ONEBODY, cubic box.
 * All pairs are scanned (no cell list): meant for the small systems of such loops, N <= SE_NOALLOC_MAX_N.
 * Arguments: N particles; L box edge; xi splitting parameter; r_c cutoff, 0 < r_c <= L/2; eta0 viscosity;
 * pos [N][3], radii [N], F [N][3], T [N][3], S [N][5] DEVICE pointers, read only, caller-owned, layout as in
 * far_mobility_apply; U [N][3], Omega [N][3], E [N][5] DEVICE pointers, overwritten; cuda_stream a cudaStream_t (NULL = legacy
 * default stream); err / err_len an optional caller buffer that receives the error text (may be NULL / 0).
 * Scratch: the packed copies and the per-particle sums live in ONE static device array inside the library,
 * SE_NOALLOC_MAX_N * 29 doubles = 1.9 MB, held by every GPU that loads the library until the process exits.  Every call on a
 * device shares it: calls that overlap on the GPU (different streams, different host threads) RACE -- order them on one stream
 * or with events.  It keeps the last call's contents; nothing in it has to start at zero (every field read is written first by
 * the same call).  The first call on each device asks the runtime for the array's device address (no allocation); the launch
 * itself is three kernels on the caller's stream and returns without synchronising.
 * Errors: SE_ERR_INVALID_ARG for N < 1, N > SE_NOALLOC_MAX_N (text says so), a parameter out of range or a NULL pointer (nothing
 * is launched); SE_ERR_CUDA when the address cannot be had or a launch fails.  Calls no cudaMalloc, cudaFree, cuFFT. */
#define SE_NOALLOC_MAX_N 8192
se_status far_mobility_real_noalloc(int64_t N, double L, double xi, double r_c, double eta0, const double *pos, const double *radii,
                                    const double *F, const double *T, const double *S, double *U, double *Omega, double *E,
                                    void *cuda_stream, char *err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* SE_MOBILITY_H */
