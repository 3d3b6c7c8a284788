/* mbhl.h - C ABI of the B200-native batched LISA massive-black-hole-binary log-likelihood.
 *
 * Implements the likelihood hot path of arXiv:2005.01827 (section II.A):
 *   one-time upload of the data stream and noise PSD
 *   per call, for each parameter set ("walker"):
 *     PhenomHM amplitude/phase of 6 modes on a sparse grid      (eq. 5)
 *     t_lm(f), frequency bounds                                 (eq. 6)
 *     fast frequency-domain LISA response, TDI A/E/T            (eqs. 7-10)
 *     cubic-spline coefficients of the sparse smooth functions
 *     interpolation to the dense Fourier grid, mode sum, PSD-weighted inner products,
 *     logL = -1/2 <d-h|d-h> = <d|h> - 1/2 <h|h> - 1/2 <d|d>     (eqs. 2, 3, 11)
 * All arithmetic is fp64 and runs in hand-written sm_100a CUDA kernels; there is no CPU path.
 * CAVEAT: the model's STRUCTURE is PhenomD/PhenomHM as published, its fit NUMBERS are not: the paper prints none and the
 * cited tables are not available offline, so model_data/phenomhm_table.csv holds smooth surrogate stand-ins (provenance tag
 * per entry).  logL will not agree with a real PhenomHM pipeline until that data file is replaced (reading G1).
 * The readings of the paper that fix what is silent or ambiguous are listed in DESIGN.md section 4.
 *
 * Conventions common to all calls
 *   - Return value: 0 (MBHL_OK) or a negative MBHL_E* code; never throws, never aborts.
 *     mbhl_last_error(ctx) gives a message for the last failing call on that context.
 *   - "device pointer" = memory on the context's CUDA device (e.g. torch.Tensor.data_ptr()).
 *   - Hot-path calls (mbhl_loglike*, mbhl_template, mbhl_sparse) are ASYNCHRONOUS on the
 *     context's stream; outputs are valid after the caller synchronises that stream.
 *   - A context is not thread-safe; several contexts may coexist.
 *   - Parameter vector, 11 doubles per walker, row-major [B][11]:
 *       0 M_T   total mass, detector frame [solar masses]
 *       1 q     mass ratio; any q > 0 is accepted, q and 1/q are the same binary (reading G15)
 *       2 a1    dimensionless aligned spin of the HEAVIER body, |a1| <= 1
 *       3 a2    dimensionless aligned spin of the lighter body, |a2| <= 1
 *       4 D_L   luminosity distance [Gpc]
 *       5 phi_ref  reference phase [rad]
 *       6 iota  inclination [rad]
 *       7 lambda   ecliptic longitude, SSB frame [rad]
 *       8 beta  ecliptic latitude, SSB frame [rad]
 *       9 psi   polarisation angle [rad]
 *      10 t_ref reference time [s]; t_coal = t0 + t_ref, t = 0 is the start of the data
 *   - Per-walker domain errors are not call errors: a walker with a non-finite parameter,
 *     M_T <= 0, D_L <= 0, q <= 0, |a1| > 1 or |a2| > 1 gets logL = -inf and <d|h> = <h|h> = 0;
 *     a valid walker whose modes all fall outside the grid gets logL = -1/2 <d|d>.  Never NaN.
 *   - Mode order everywhere: (2,2),(3,3),(4,4),(2,1),(3,2),(4,3).
 *   - Splined quantities per (walker, mode), Q = 8, in this order (reading G8):
 *       0 A_lm [strain*s]; 1 Phi_lm = phi_lm + phi_Doppler without the linear term -2 pi f t_coal;
 *       2,3 Re,Im That^A; 4,5 Re,Im That^E; 6,7 Re,Im That^T.
 */
#ifndef MBHL_H
#define MBHL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MBHL_OK        0
#define MBHL_EINVAL   -1   /* null pointer, bad size, non-uniform / non-increasing / non-positive grid   */
#define MBHL_ENOMEM   -2   /* device or host allocation failed                                           */
#define MBHL_ECUDA    -3   /* CUDA runtime error, text in mbhl_last_error                                */
#define MBHL_ENOWS    -4   /* caller-supplied workspace too small for this batch                         */

/* Coordinates a walker row may be given in (mbhl_loglike_coords, mbhl_unpack_coords, mbhl_pt_init) */
#define MBHL_COORDS_PHYSICAL      0   /* the 11 physical SSB-frame parameters listed above                            */
#define MBHL_COORDS_SAMPLED       1   /* the sampler's coordinates: (ln M_T, q, a1, a2, ln D_L, phi_ref,
                                         cos iota, lambda, sin beta, psi, ln t_ref), sky/polarisation/time in the SSB   */
#define MBHL_COORDS_SAMPLED_LISA  2   /* the same with (lambda, sin beta, psi, ln t) in the LISA frame:
                                         what the paper's sampler hands over.  Reading G20 of DESIGN.md: frame of the
                                         constellation at the orbital phase Omega_0 (t0 + t_L), t_L = arrival time of the
                                         wavefront at the constellation centre                                          */

#define MBHL_NPARAM   11
#define MBHL_NMODE     6
#define MBHL_NQ        8

typedef struct mbhl_ctx mbhl_ctx;     /* opaque; owned by the library, released by mbhl_free */

typedef struct mbhl_config {
    int32_t  sparse_points;  /* S, knots per mode, 8 <= S <= 2048 (one CTA's shared memory holds a mode's knots
                                and right-hand sides); 0 = default 1024 ("~2^10")                    */
    uint32_t mode_mask;      /* bit i enables mode i of the order above; 0 = all six                     */
    double   t0;             /* t_coal = t0 + t_ref                                       */
    int64_t  max_batch;      /* workspace for this many walkers is allocated at init; 0 = grow on demand.  With
                                max_batch >= B (or a caller workspace) mbhl_loglike* allocates nothing and never
                                synchronises: the call may be captured in a CUDA graph on the context's stream  */
    int32_t  device;         /* CUDA device ordinal                                                      */
    void*    stream;         /* cudaStream_t all work is enqueued on; NULL = legacy default stream       */
} mbhl_config;

/* One-time setup.  freqs[N]: strictly increasing, uniform (relative tolerance 1e-6 on the
 * spacing), freqs[0] > 0, N >= 4.  data_AET[3][N][2]: (Re, Im) of d^A, d^E, d^T.  psd_AET[3][N]: one-sided
 * noise PSD; bins with S_n <= 0 or non-finite get weight 0 (reading G6).  The three arrays may be host or
 * device pointers (detected); they are copied/transformed into library-owned device buffers
 * (w = 4 df / S_n with df = (f[N-1]-f[0])/(N-1), w*d, and <d|d>), so the caller may free them afterwards.
 * cfg == NULL means all defaults on device 0.  On success *out holds the new context.                   */
int mbhl_init(mbhl_ctx** out, const double* freqs, int64_t N, const double* data_AET,
              const double* psd_AET, const mbhl_config* cfg);

/* logL[b] for params[b][11], b < B (eq. 2).  params, logL: device pointers, caller-owned.  B >= 0.       */
int mbhl_loglike(mbhl_ctx* ctx, const double* params, int64_t B, double* logL);

/* Same, also returning <d|h> and <h|h> (either may be NULL); logL = d_h - h_h/2 - <d|d>/2.               */
int mbhl_loglike_parts(mbhl_ctx* ctx, const double* params, int64_t B,
                       double* d_h, double* h_h, double* logL);

/* Host-buffer convenience for end-to-end use: params_host[B][11] and logL_host[B] are HOST pointers
 * (pinned memory makes the copies asynchronous); the call enqueues H2D, the hot path and D2H on the
 * context's stream and synchronises it before returning.                                               */
int mbhl_loglike_host(mbhl_ctx* ctx, const double* params_host, int64_t B, double* logL_host);

/* Template h^{A,E,T} of each walker on freqs_out[Nout] (device pointer; NULL = the init grid, Nout ignored),
 * written to out_AET[B][3][Nout][2] (device).  direct = 0: the spline path the likelihood uses;
 * direct = 1: waveform + response evaluated at every bin (no spline).  A mode contributes only inside its
 * band [f_lo, f_hi] (no extrapolation).  Testing / injection aid (PAPER.md:171 stores this; the
 * likelihood path never does).                                                                          */
int mbhl_template(mbhl_ctx* ctx, const double* params, int64_t B, const double* freqs_out,
                  int64_t Nout, double* out_AET, int32_t direct);

/* Sparse stage only (steps a1-a5).  Any output may be NULL.  Device pointers.
 *   knots[B][6][S]      log-spaced knots f_s [Hz]; all 0 for an inactive mode
 *   y[B][6][8][S]       the Q = 8 smooth functions at the knots (Phi in radians)
 *   coef[B][6][S-1][8][4]  per interval (y_j, s_j, c_j, d_j): p = y_j + s_j u + c_j u^2 + d_j u^3, u = f - f_j.
 *                       The Phi row is stored in CYCLES (Phi / 2 pi) with y_j reduced into [-1/2, 1/2].    */
int mbhl_sparse(mbhl_ctx* ctx, const double* params, int64_t B, double* knots, double* y, double* coef);

/* Workspace the hot path needs for a batch of B (bytes).                                                 */
size_t mbhl_workspace_bytes(const mbhl_ctx* ctx, int64_t B);
/* Optional caller-owned workspace (device pointer, 256-byte aligned); once set the library performs no
 * device allocation in the hot path and returns MBHL_ENOWS if it is too small.  NULL returns to internal.*/
int mbhl_set_workspace(mbhl_ctx* ctx, void* dev_ptr, size_t bytes);

/* ---- Sampler-side steps next to the likelihood (section II.B) -------------------- */

/* Per-mode inner products (Table III :292-300): every mode evaluated in isolation against the
 * data.  d_h[B][6] = <d|h_lm>, h_h[B][6] = <h_lm|h_lm> (optimal SNR of the mode alone = sqrt);
 * either may be NULL.  Device pointers; mode order as above; a mode disabled at init gives 0.               */
int mbhl_mode_products(mbhl_ctx* ctx, const double* params, int64_t B, double* d_h, double* h_h);

/* logL for walkers given in the coordinates `coords` (MBHL_COORDS_*).  For the two sampled forms every component is
 * uniform between the bounds of Table I and a walker outside that box gets logL = -inf (zero prior);
 * with MBHL_COORDS_SAMPLED_LISA the box applies to the LISA-frame values.  The conversion to physical SSB parameters
 * (exp / acos / asin, LISA -> SSB rotation and arrival-time shift) runs inside the per-walker constants kernel.
 * rows[B][11], logL[B]: device pointers.  mbhl_loglike_sampled(ctx, theta, B, logL) is coords = MBHL_COORDS_SAMPLED.     */
int mbhl_loglike_coords(mbhl_ctx* ctx, const double* rows, int64_t B, int32_t coords, double* logL);
int mbhl_loglike_sampled(mbhl_ctx* ctx, const double* theta, int64_t B, double* logL);

/* The conversion alone: params_out[B][11] (device) receives the physical SSB parameters of every row (a NaN row for a
 * walker outside the prior box).  Testing aid; asynchronous on the context's stream.                                    */
int mbhl_unpack_coords(mbhl_ctx* ctx, const double* rows, int64_t B, int32_t coords, double* params_out);

/* mbhl_unpack_coords for callers that must not allocate device memory.
 * WHO THAT IS: mbhl_unpack_coords (like every hot-path call) takes its per-walker records from the context's workspace,
 * and on a context created without max_batch or a caller workspace that means a cudaMalloc inside the call.  Some callers
 * cannot afford or are not allowed that: a sampler sharing the GPU with a framework whose memory pool has already claimed
 * all free HBM (the cudaMalloc would simply fail), a job running under a fixed per-process memory quota, or a latency-critical
 * loop in which cudaMalloc / cudaFree would stall the device's other streams while they run.  For them this entry point does the same
 * conversion - the same kernel, k_walker_consts - with the kernel's scratch records (the WalkerConst and DenseWalker of every
 * row, about 2.5 KB per walker, which this call computes and then discards) placed in a fixed array that is part of the
 * library image instead of in allocated memory.  It calls no cudaMalloc, cudaFree or any allocating library routine.
 *   rows[B][11] (device, in `coords`) -> params_out[B][11] (device): physical SSB parameters, a NaN row for a walker outside
 *   the prior box - bit-for-bit what mbhl_unpack_coords writes.  Caller owns both; they must not overlap (MBHL_EINVAL).
 * LIMIT: B <= MBHL_STATIC_MAX_WALKERS per call; a larger B is refused with MBHL_EINVAL and a message naming the limit
 * (split the batch).  The array is sized for exactly that many walkers (about 2.6 MB) and every GPU on which the library
 * is loaded holds it until the process exits, whether or not this call is ever made.
 * FIRST CALL: the first call on each device looks up the array's device address (cudaGetSymbolAddress, once per device,
 * kept for the process's lifetime); that lookup may make the driver load the library's module.  Make this first call
 * during set-up, before any stream capture is begun.
 * SHARING: there is ONE array per device, shared by every context, stream and thread, and it keeps the previous call's
 * records.  Nothing in it has to start at zero - each call overwrites the records of its rows 0..B-1 before anything could
 * read them and never looks at the rest - so stale contents are harmless.  But two calls whose kernels can overlap on the
 * same GPU (different streams, different contexts, different host threads) write the same records and race: keep calls on one
 * device ordered on one stream, or synchronise between them.  Asynchronous on the context's stream.                      */
#define MBHL_STATIC_MAX_WALKERS 1024
int mbhl_unpack_coords_static(mbhl_ctx* ctx, const double* rows, int64_t B, int32_t coords, double* params_out);

/* Parallel-tempered affine-invariant ensemble: n_temps rungs with inverse temperatures
 * betas[t] (host pointer; beta = 0 is T = infinity, :222), n_walkers (even) walkers per rung in the sampler's
 * coordinates, theta0[n_temps][n_walkers][11] (host or device pointer, copied).  One step = for each half of the
 * ensemble a stretch move of every walker of that half against a partner drawn from the other half of its
 * rung (eqs. 14-16 with parameter stretch_a, 1.15 in the paper) - the proposals of all rungs go through the
 * likelihood hot path as ONE batch - then one sweep of swaps between adjacent rungs from the hottest pair
 * down (eq. 17).  The target of rung t is prior x L^beta_t with the uniform prior of Table I (:211).  Random
 * numbers: Philox4x32-10 keyed by seed, counter (walker, step, stream), so a run is reproducible.  The
 * ensemble lives on the context's device and stream; nothing returns to the host between steps.
 * coords = MBHL_COORDS_SAMPLED or MBHL_COORDS_SAMPLED_LISA (the frame the walkers live in).  Every starting walker must
 * lie inside the prior box and have a finite logL (else MBHL_EINVAL): a walker at logL = -inf could never move on the
 * beta = 0 rung.  n_temps * n_walkers <= 65535.  The context must outlive the ensemble.                     */
typedef struct mbhl_pt mbhl_pt;
int  mbhl_pt_init(mbhl_ctx* ctx, mbhl_pt** out, const double* theta0, const double* betas, int32_t n_temps,
                  int32_t n_walkers, uint64_t seed, double stretch_a, int32_t coords);
int  mbhl_pt_step(mbhl_pt* pt, int32_t n_steps);                  /* asynchronous on the context's stream   */
/* Copies the ensemble out and synchronises: theta[n_temps][n_walkers][11], logL[n_temps][n_walkers] (host or
 * device), accepted moves per rung n_accept[n_temps] and accepted swaps n_swap[n_temps-1] (host).  Any may be NULL. */
int  mbhl_pt_state(mbhl_pt* pt, double* theta, double* logL, int64_t* n_accept, int64_t* n_swap);
void mbhl_pt_free(mbhl_pt* pt);

/* Heterodyned ("relative binning") likelihood - an accuracy-controlled variant of the hot path ("we may
 * test different approximations in our GPU implementation"; definition: DESIGN.md section 10, reading H1).
 * mbhl_het_init evaluates the spline template's per-mode phase of the reference parameters params_ref[11] (device
 * pointer, physical SSB) on the context's grid and accumulates, once, the summary data of the coarse bins
 * [edges[b], edges[b+1]) (edges: HOST pointer, n_coarse + 1 bin indices, edges[0] = 0 < ... < edges[n_coarse] = N; the
 * library refines them by the reference's band edges, so that every mode is in band throughout a coarse bin or absent).
 * mbhl_het_loglike then evaluates walkers from the summary data: per walker the sparse stage (a1-a5) plus
 * 3 n_coarse spline evaluations per mode, instead of one per fine bin.  The envelope A That exp(i (theta - theta_ref))
 * is taken piecewise parabolic on the coarse bins (values at a bin's first, centre and last frequency): exact for one
 * fine bin per coarse bin; otherwise the error of the sums falls at least with the cube of the coarse bin width (with its fourth power on bins that hold no band edge and no region boundary of the model: pinned on the oracle in tests/test_oracle_heterodyne.py); accurate for walkers whose phase stays within a fraction of a cycle of the reference's across a
 * coarse bin (the bulk of a posterior).  The band of a mode is taken to be the reference's, and a coarse bin that the walker's own band of that mode does not reach contributes nothing, as in mbhl_loglike; no spline is extrapolated.  d_h, h_h, logL [B]: device
 * pointers, any may be NULL.  Asynchronous on the context's stream EXCEPT when a batch is larger than any this handle has seen:
 * its partial-sum buffer ([B][coarse-bin groups][2] doubles) then grows, which synchronises the stream and calls cudaFree /
 * cudaMalloc; call once with the largest batch during set-up to keep later calls free of both.  The context must outlive the handle. */
typedef struct mbhl_het mbhl_het;
int  mbhl_het_init(mbhl_ctx* ctx, mbhl_het** out, const double* params_ref, const int64_t* edges, int32_t n_coarse);
int  mbhl_het_loglike(mbhl_het* het, const double* params, int64_t B, double* d_h, double* h_h, double* logL);
void mbhl_het_free(mbhl_het* het);

/* Noise realisation for fabricating data streams (eq. 12; reading G5 of DESIGN.md): for each channel
 * and bin Re, Im ~ N(0, S_n / (4 df)) independent (the circular Gaussian that eq. 12's "normal modulus, uniform phase"
 * approximates), drawn by Box-Muller from Philox4x32-10 with key = seed and counter (bin, channel, 3, 0).  psd_AET[3][N]
 * and out_AET[3][N][2] are device pointers on the current device; bins with S_n <= 0 or non-finite get 0.
 * Needs no context; asynchronous on `stream` (cudaStream_t, NULL = default stream).  N <= 2^31.            */
int mbhl_noise(void* stream, const double* psd_AET, int64_t N, double df, uint64_t seed, double* out_AET);

/* Introspection. */
double  mbhl_data_norm(const mbhl_ctx* ctx);        /* <d|d> computed at init                            */
int64_t mbhl_num_bins(const mbhl_ctx* ctx);
int32_t mbhl_sparse_points(const mbhl_ctx* ctx);
int64_t mbhl_launch_count(const mbhl_ctx* ctx);     /* kernels this context has launched so far          */
/* Work counters of the last mbhl_loglike* call (device -> host copy, synchronises the stream):
 * pairs = sum over walkers and modes of in-band bins, bins = sum over walkers of bins covered by >= 1 mode. */
int mbhl_last_work(mbhl_ctx* ctx, int64_t* pairs, int64_t* bins);

/* What the fused dense kernel EXECUTED in the last mbhl_loglike* call (counted in the kernel, one tally per warp), for
 * the roofline numerator: counts[0] calls of the uniform-record evaluator, counts[1] of its gated form, counts[2] of the
 * per-bin-record evaluator - each call evaluates one mode at 4 bins on all 32 lanes of a warp, in band or not -,
 * counts[3] single (lane, bin, mode) evaluations of the global per-bin path, counts[4] inner-product epilogues (each
 * covers one walker at the 128 bins of a warp).  With slices (B > 32768) the counts are those of the last slice.
 * Synchronises the stream.                                                                                          */
int mbhl_last_dense_work(mbhl_ctx* ctx, int64_t counts[5]);

/* Optional per-stage device timing.  When enabled, mbhl_loglike* records CUDA events on the context's stream
 * around its five stages; mbhl_stage_times synchronises the stream, returns the MEAN milliseconds per stage
 * over the calls made since the previous mbhl_stage_times / enable (at most the last 64) and resets the
 * count: ms[0] per-walker constants, ms[1] the fused sparse kernel (PhenomHM + response at the knots + spline
 * coefficients), ms[2] = 0 (kept for layout), ms[3] fused dense kernel, ms[4] final reduction (mbhl_sparse is timed too,
 * with ms[3] = ms[4] = 0).  Returns MBHL_EINVAL if timing is off or no call was made.                        */
int mbhl_enable_stage_timing(mbhl_ctx* ctx, int32_t on);
int mbhl_stage_times(mbhl_ctx* ctx, double ms[5]);

/* MEASUREMENT AID, not part of the method: FP64 DFMA-chain probe used by bench.py to measure the roofline denominator: each of blocks*threads threads runs
 * iters*8 dependent-chain DFMAs (8 independent chains); sink is a device pointer to >= 1 double.
 * Asynchronous on `stream`.  FLOPs = 2 * blocks * threads * iters * 8.                                   */
int mbhl_dfma_probe(void* stream, int32_t blocks, int32_t threads, int64_t iters, double* sink);

const char* mbhl_strerror(int code);
const char* mbhl_last_error(const mbhl_ctx* ctx);
void mbhl_free(mbhl_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MBHL_H */
