/*
 * sfft.h -- C ABI of libsfft_b200: the data-parallel hot path of SFFT image differencing
 * (arXiv 2109.09334, "Image Subtraction in Fourier Space") for NVIDIA B200 (sm_100a).
 *
 * Citations are "PAPER.md:<line>" (the paper's text) plus the equation; "DESIGN g#" refers
 * to a reading of a garbled or silent passage listed in DESIGN.md.
 *
 * Problem (Eqs. 1-12).  Given a reference image R and a science image S,
 * both N0 x N1 = H x W, find the coefficients of
 *     D(x,y) = S(x,y) - sum_{t,(a,b)} a_{t,ab} (R^t o K_ab)(x,y) - sum_s b_s T'_s(x,y)       (Eq. 12)
 * that minimise sum D^2, where o is circular convolution, R^t = T_t R, K_00 = delta,
 * K_ab = delta(u-a,v-b) - delta(u,v) for (a,b) != (0,0), |a|,|b| <= w, L = 2w+1 (Eqs. 3-4),
 * and T_t / T'_s are spatial weight functions of the kernel / background:
 *   SFFT_BASIS_POLY    monomials u_x^i u_y^j, i+j <= DK (resp. DB)        (Eqs. 2, 6; DESIGN g8)
 *                      of the normalised coordinates u_x = (2x+1)/H - 1, u_y = (2y+1)/W - 1
 *   SFFT_BASIS_BSPLINE tensor products B_i(v_x) B_j(v_y) of cubic B-splines on a clamped
 *                      knot vector with DK (resp. DB) uniform interior knots per axis,
 *                      v_x = (x+0.5)/H, v_y = (y+0.5)/W                    (Eqs. 8-9; DESIGN g13)
 *
 * Layout and indices.  Images are row-major double [x][y], x in [0,H) slow, y in [0,W) fast;
 * with nbatch > 1 they are [b][x][y] (independent pairs).  Lag index a = (alpha+w)*L + (beta+w),
 * centre a0 = w*L+w.  Unknown k = t*L*L + a (kernel) or F_K*L*L + s (background);
 * n = F_K*L*L + F_B.  POLY terms t <-> (i,j): i = 0..D outer, j = 0..D-i inner;
 * BSPLINE terms t = i*(D+4) + j.  Coefficients are the real-space a-ring of the paper
 * (the paper's a = N0 N1 a-ring), with the photometric scale free (DESIGN g9).
 *
 * All pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The caller owns every
 * buffer, including the workspace; the plan owns only small constant tables.  Calls enqueue
 * work on the plan's CUDA stream and return without synchronising unless stated.  Every call
 * returns an SFFT_* status; nothing throws or aborts.  There is no CPU fallback: without a
 * CUDA device every compute call returns SFFT_ERR_CUDA.  A plan belongs to the CUDA device that was
 * current when it was created; calling it with another device current returns SFFT_ERR_STATE.
 */
#ifndef SFFT_H_
#define SFFT_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sfft_plan sfft_plan; /* opaque host-side handle */

enum { SFFT_BASIS_POLY = 0, SFFT_BASIS_BSPLINE = 1 };

enum {
    SFFT_OK = 0,
    SFFT_ERR_INVALID_ARG = 1, /* bad size / null pointer / unsupported shape                */
    SFFT_ERR_STATE = 2,       /* call order violated (e.g. solve before build)              */
    SFFT_ERR_WORKSPACE = 3,   /* workspace missing or too small                              */
    SFFT_ERR_CUDA = 4,        /* CUDA runtime error (message via sfft_last_cuda_error)       */
    SFFT_ERR_NOT_SPD = 5      /* normal matrix not positive definite (rank-deficient input)  */
};

/* Create a plan for H x W images, L x L kernel (L odd), spatial orders DK / DB, given basis.
 * POLY: DK, DB = total polynomial degree.  BSPLINE: DK, DB = number of uniform interior knots.
 * Restrictions (INVALID_ARG otherwise): 32 <= H <= 8192, 64 <= W <= 8192, W even; L odd, 1 <= L <= 33,
 * 2L-1 <= min(H, W); DK, DB in [0, 8].  Frames whose H or W is not a power of two (NEXT-4; true CCD frames such as
 * 2046 x 4094) additionally need W <= 4096 when W is not a power of two, the polynomial basis and
 * DK <= 2: their rows are transformed by a chirp-z (Bluestein) DFT (forward and inverse) and the lag correlation
 * takes the sectioned route; sfft_decorrelate needs tiles that divide the frame.
 * Builds constant tables on the host and uploads them (synchronous). */
int sfft_plan_create(sfft_plan **out, int H, int W, int L, int DK, int DB, int basis);

/* NEXT-4, rectangular kernels (the delta basis spans L0 x L1 pixels, |alpha| <= (L0-1)/2 along x and
 * |beta| <= (L1-1)/2 along y; L0, L1 odd, 1 <= L0, L1 <= 33, other restrictions as above with L = max(L0, L1)).
 * Every layout of this header keeps the enclosing SQUARE L = max(L0, L1): n = F_K*L*L + F_B, lag index
 * a = (alpha+w)*L + (beta+w) with w = (L-1)/2, and the coefficients outside the rectangle are fixed at zero
 * (sfft_solve writes them as 0; vectors given to sfft_subtract are used as they are).  The system that is
 * assembled and solved holds only the free unknowns: sfft_plan_num_solved() = F_K*L0*L1 + F_B of them (fewer under
 * the constant photometric ratio), in the order of the full layout with the fixed entries removed - for L0 != L1
 * that is exactly the order t*L0*L1 + (alpha+w0)*L1 + (beta+w1) of the rectangular model.  The lag tables are
 * formed for the enclosing square, so the cost is that of an L x L kernel.  sfft_plan_create(.., L, ..) is
 * sfft_plan_create_rect(.., L, L, ..). */
int sfft_plan_create_rect(sfft_plan **out, int H, int W, int L0, int L1, int DK, int DB, int basis);

/* Number of independent pairs processed per call (default 1).  Must precede set_workspace. */
int sfft_plan_set_batch(sfft_plan *plan, int nbatch);

/* CUDA stream (cudaStream_t cast to void*; NULL = legacy default stream). */
int sfft_plan_set_stream(sfft_plan *plan, void *cuda_stream);

/* NEXT-1, constant photometric ratio (PAPER.md:121, 264 -ConstPhotRatio): on = 1 constrains the kernel integral
 * sum_t a_{t,00} T_t(x,y) to a constant (POLY: a_{t,00} = 0 for t >= 1; BSPLINE: all a_{t,00} equal), leaving
 * sfft_plan_num_solved() = (free unknowns) - (F_K - 1) unknowns in the system returned by sfft_get_system (order of
 * the full layout with the centre entries of t >= 1 removed).  Coefficient vectors keep the full layout of n entries,
 * the constrained ones filled in.  Default 0 (BASELINE.json's unknown counts).  Call before sfft_build_system. */
int sfft_plan_set_const_phot_ratio(sfft_plan *plan, int on);
int sfft_plan_num_solved(const sfft_plan *plan);

/* Route of the x-direction lag correlation (steps a3+a4): 0 = chosen by the plan (default), 1 = direct lag sums
 * on the FP64 tensor cores, 2 = sectioned (overlap-save) correlation with 64-point FFTs along x, available for
 * polynomial bases with at most 8 column sequences (F_K + 1 <= 8), SFFT_ERR_INVALID_ARG otherwise.  Both routes
 * evaluate the same sums (App. B) and agree to rounding (bit for bit in their x-weights only when H
 * is a power of two); the setter exists so that parity tests and benchmarks can
 * run either on the same input.  Invalidates the workspace (call before sfft_plan_workspace_bytes). */
int sfft_plan_set_corr_route(sfft_plan *plan, int route);

/* n = F_K*L*L + F_B (Eq. 18's dimension), or -1 for a null plan. */
int sfft_plan_num_unknowns(const sfft_plan *plan);
int sfft_plan_num_kernel_terms(const sfft_plan *plan);     /* F_K */
int sfft_plan_num_background_terms(const sfft_plan *plan); /* F_B */

/* Bytes of device workspace the plan needs for its current batch size (build / solve / subtract on device
 * pointers; the image staging area of the host-buffer entry points is a separate buffer, see below). */
size_t sfft_plan_workspace_bytes(const sfft_plan *plan);

/* Lend a device buffer (>= workspace_bytes, 256-byte aligned) to the plan.  The caller keeps
 * ownership and must keep it alive until the plan is destroyed or another buffer is set.  Enqueues a
 * clearing of part of the buffer on the plan's stream (set the stream first), and the plan relies on the contents
 * from then on: while the buffer is lent the caller must not write to it (lend it again with this call after using
 * it for something else). */
int sfft_plan_set_workspace(sfft_plan *plan, void *d_ws, size_t bytes);

/* Steps a1-a5: assemble the normal system of Eq. 18 in real-space scaling,
 * M = Phi^T Phi, rhs = Phi^T S, from the pair (d_R, d_S), each [nbatch][H][W] double.
 * Every block is a cross-correlation of weighted images evaluated by FFT and read at the
 * kernel-lag offsets only (App. B).  Inputs are not modified.
 * Part of the work (the image-by-basis-function moments) is enqueued on a stream the plan owns, forked from
 * and joined back into the plan's stream with events: ordering on the plan's stream is all a caller sees. */
int sfft_build_system(sfft_plan *plan, const double *d_R, const double *d_S);

/* Device pointers to the assembled system (valid until the next build): M is [nbatch][ns][ld] row-major,
 * FULL symmetric (both triangles), ld = ns = sfft_plan_num_solved() (= n unless the photometric ratio is
 * constrained); rhs is [nbatch][ns].  For parity tests. */
int sfft_get_system(const sfft_plan *plan, const double **d_M, const double **d_rhs, int *ld);

/* Device pointer to the lag tables of the last build, for parity tests.  which: 0 = Omega
 * [npairs][2L-1][2L-1] over pairs (tb <= t) in row-major pair order, 1 = Theta [F_K][L][L],
 * 2 = Lambda [F_K][F_B][L][L], 3 = Delta [F_B].  *d_table points at the table of batch entry 0; the
 * same table of batch entry b starts *batch_stride doubles further per entry.  count receives the number
 * of doubles of the table (per batch entry).  count and batch_stride may be NULL. */
int sfft_get_lag_table(const sfft_plan *plan, int which, const double **d_table, size_t *count, size_t *batch_stride);

/* Step a6: solve M c = rhs (Jacobi-scaled blocked FP64 Cholesky; DESIGN g11) and write
 * c to d_coef [nbatch][n].  A diagonal entry that is not positive and finite, or a pivot of the
 * Jacobi-scaled matrix (unit diagonal) that is not finite or falls below 64 n eps (eps = 2^-52: the level
 * at which a pivot is rounding noise of the assembled entries, i.e. the system is numerically
 * rank-deficient), raises a device flag reported by sfft_plan_status as SFFT_ERR_NOT_SPD; d_coef is then
 * undefined.  The back substitution is a chain of CTAs that wait for one another through global memory; each takes
 * its place in the chain from a counter when it starts running, so it only waits for CTAs that have started
 * already and the call cannot deadlock on the order in which the grid is dispatched. */
int sfft_solve(sfft_plan *plan, double *d_coef);

/* Steps a7-a8: D = S - sum_t sum_ab k_{t,ab} R^t((x-a)%H,(y-b)%W) - sum_s b_s T'_s  (Eqs. 1, 12)
 * with k the delta-basis coefficients folded back to pixel kernels (Eqs. 3-4).  (d_R, d_S)
 * may differ from the fitted pair (fit on the masked pair, apply to the
 * original).  d_D [nbatch][H][W] may alias d_S; no other aliasing.
 * Two routes, chosen by the plan from its sizes: the direct tensor-core contraction, or (wide
 * kernels on rows of >= 1024 pixels) a FIR filter along x on the row spectra followed by one
 * inverse row transform.  The second route needs the row spectra of d_R: by default it transforms
 * d_R again on every call (whatever was passed to sfft_build_system); see sfft_plan_set_reuse_spectra
 * for the opt-in that skips this.  It overwrites the workspace slot holding the row spectrum of S. */
int sfft_subtract(sfft_plan *plan, const double *d_coef, const double *d_R, const double *d_S, double *d_D);

/* Opt-in for the Fourier-route subtract: on = 1 is the caller's PROMISE that every following sfft_subtract is
 * given, as d_R, an image with the same contents as the d_R of the last sfft_build_system (the unmasked flow:
 * fit and apply on the same pair); the row spectra computed by that build are then reused instead of
 * transforming d_R again.  Pointer values play no role in either mode.  Default 0: always transform again,
 * which is what the paper's masked flow needs (fit on the masked pair, apply to the original).
 * The host-buffer entry points below fit and apply on the same staged pair and always reuse. */
int sfft_plan_set_reuse_spectra(sfft_plan *plan, int on);

/* NEXT-2, crowded-flavor preprocessing (reading DESIGN g21): build the masked pair the fit runs on.
 *   seed = d_R >= sat_R or d_S >= sat_S (one joint mask for the pair), mask = seed grown by rd pixels (square
 *   (2 rd + 1)^2 window), every masked pixel of an image replaced by the mean of that image's unmasked pixels in the
 *   (2 rb + 1)^2 window around it (by the mean of all its unmasked pixels if that window holds none), unmasked pixels
 *   copied; indices wrap around.  d_Rm, d_Sm: [nbatch][H][W] double, may alias d_R, d_S (in place); d_mask:
 *   [nbatch][H][W] unsigned char, 1 = masked.  0 <= rd <= 64, 1 <= rb <= 128.  Needs the workspace (its spectrum
 *   area is used as scratch, so call it before sfft_build_system, not between build and subtract).
 * The paper's flow is then sfft_build_system(d_Rm, d_Sm) -> sfft_solve -> sfft_subtract(d_R, d_S). */
int sfft_mask_fill(sfft_plan *plan, const double *d_R, const double *d_S, double sat_R, double sat_S, int rd, int rb,
                   double *d_Rm, double *d_Sm, unsigned char *d_mask);

/* The same mask/fill for ONE pair (nbatch = 1), for callers that have no way to obtain device memory for the
 * library: no plan, no workspace, and no cudaMalloc / cudaFree / allocating library routine anywhere in the call.
 * Who needs this: a process whose device memory was all handed to one pool at start-up (a late cudaMalloc there
 * fails, or falls outside the pool's accounting), and a loop that must never stall (cudaMalloc and cudaFree
 * synchronise the whole device).  sfft_plan_create uploads tables into memory it allocates and sfft_mask_fill wants a
 * lent workspace, so neither serves such a caller; this call takes the five images and nothing else.
 *   Its scratch (row-grown seed flags, one byte per pixel, plus 32 KiB of partial sums) lives in an array that is part
 *   of the library image: SFFT_STATIC_MAX_PIXELS + 32768 bytes (16 MiB + 32 KiB) of device memory on EVERY GPU on which
 *   the process uses this library, held from the moment the library's device code is loaded there until the process
 *   exits, whether or not this call is ever made.
 *   Limits: 1 <= H, W <= 16384 and H*W <= SFFT_STATIC_MAX_PIXELS (4096 x 4096, which covers the 2046 x 4094 CCD
 *   frame); anything larger is refused with SFFT_ERR_INVALID_ARG and a message naming the limit
 *   (sfft_static_last_error).  rd, rb, sat_*, the pointer roles, aliasing and layout are those of sfft_mask_fill,
 *   and so is the result, bit for bit (the same kernels run).  Any H and W are accepted (indices wrap by modulo);
 *   with W even and the four images 16-byte aligned (the mask 2-byte aligned) the faster two-pixels-per-thread kernels
 *   run, otherwise one-pixel-per-thread forms of them (same mask; the global-mean fallback may differ in its last bit).
 *   Set-up: the first call on each device looks up the device address of the scratch array (once per device, cached;
 *   the device that is current at the call is the one used, and d_* and cuda_stream must belong to it).  That
 *   look-up may make the CUDA runtime load the library's device code, so issue the first call on a device ahead of
 *   any stream capture and ahead of the section that must not stall.
 *   Sharing: every call on a device uses the same scratch, and the scratch keeps the previous call's contents.
 *   Nothing in it has to start at zero: each call writes every entry it later reads (H*W flags, 3552 partial sums,
 *   2 means) before reading it, so no clearing pass is run.  Two calls that can overlap on the GPU (different
 *   streams, or different host threads without ordering) race on it and both results are garbage: order them on one
 *   stream or with events.
 *   cuda_stream: cudaStream_t cast to void* (NULL = legacy default stream).  Work is enqueued, not synchronised.
 * sfft_static_last_error: message of the last failing sfft_mask_fill_static call of the calling thread ("" if none). */
#define SFFT_STATIC_MAX_PIXELS (4096L * 4096L)
int sfft_mask_fill_static(const double *d_R, const double *d_S, int H, int W, double sat_R, double sat_S, int rd,
                          int rb, double *d_Rm, double *d_Sm, unsigned char *d_mask, void *cuda_stream);
const char *sfft_static_last_error(void);

/* NEXT-3, noise decorrelation of a difference image (App. C; readings DESIGN g22).  With
 *   D = sum_j S_j (*) G_j - [sum_i R_i (*) H_i] (*) K                                            (C17)
 *   Q0^ = sqrt( sigma_D^2 / { sum_j varS_j |G_j^|^2 + sum_i varR_i |K^|^2 |H_i^|^2 } )           (C20)
 * and Q normalised to unit kernel sum, d_Ddc = D (*) Q, segment by segment: the frame
 * is cut in square tiles of `tile` pixels (a power of two in [32, 512] dividing H and W, >= L), K is the fitted
 * kernel of d_coef frozen at each tile's centre pixel (tile/2, tile/2 of the tile), and every tile is convolved
 * circularly with its own Q.  G_j (nS kernels, LG x LG, row-major, centred, LG odd <= tile) and H_i (nR kernels,
 * LH x LH) are the PSF-homogenisation kernels of the co-added science / reference images, already divided by the
 * number of images as in the paper; varS / varR their background noise variances.  For a plain pair pass
 * nS = nR = 1, LG = LH = 1, G = H = {1.0}.  h_* are HOST arrays (read before the call returns).  d_D, d_Ddc:
 * [nbatch][H][W] double, may alias.  Uses the spectrum area of the workspace as scratch (SFFT_ERR_WORKSPACE if it is
 * too small for the tile size), so a following Fourier-route sfft_subtract transforms its reference again. */
int sfft_decorrelate(sfft_plan *plan, const double *d_coef, const double *d_D, double *d_Ddc, int tile,
                     int nS, const double *h_varS, int LG, const double *h_G,
                     int nR, const double *h_varR, int LH, const double *h_H);

/* Synchronise the plan's stream and report numerical status.  On SFFT_ERR_NOT_SPD, *info =
 * batch*ns + index of the first failing pivot in the order of the solved system (ns =
 * sfft_plan_num_solved(): the reduced layout under the constant photometric ratio); otherwise
 * *info = -1.  info may be NULL. */
int sfft_plan_status(sfft_plan *plan, int *info);

/* Device staging area of the host-buffer entry points (two slots of R, S, D images and coefficients):
 * size for the current batch, and the call that lends a caller-owned device buffer (>= that size, 256-byte
 * aligned) to the plan.  Callers that only use device pointers never need it. */
size_t sfft_plan_host_staging_bytes(const sfft_plan *plan);
int sfft_plan_set_host_staging(sfft_plan *plan, void *d_buf, size_t bytes);

/* End-to-end convenience with HOST buffers: copies h_R, h_S ([nbatch][H][W]) to the device,
 * runs build -> solve -> subtract, copies D and the coefficients back, synchronises.
 * Needs the workspace and the staging area (SFFT_ERR_WORKSPACE otherwise).
 * h_D [nbatch][H][W], h_coef [nbatch][n] (either may be NULL to skip that copy). */
int sfft_run_host(sfft_plan *plan, const double *h_R, const double *h_S, double *h_D, double *h_coef);

/* The same, without the final synchronisation: the host-to-device copies, the compute and the device-to-host
 * copies are enqueued on three streams (two of them owned by the plan) over two staging slots, so that the
 * copies of one pair overlap the compute of the previous one when calls are issued back to back.  Host buffers
 * must be page-locked for the copies to be asynchronous and must stay valid (h_D, h_coef: unread) until
 * sfft_run_host_wait returns.  sfft_run_host_wait drains everything submitted and reports like sfft_plan_status. */
int sfft_run_host_async(sfft_plan *plan, const double *h_R, const double *h_S, double *h_D, double *h_coef);
int sfft_run_host_wait(sfft_plan *plan);

/* NEXT-4, FP32 storage / FP64 arithmetic: the same end-to-end calls with images stored as float on the host
 * (h_R, h_S in, h_D out: [nbatch][H][W] float; h_coef stays double).  The images are widened to double on the
 * device (exact), every step of the path computes in FP64 as before, and D is rounded to float once, on the way
 * out.  Halves the bytes crossing PCIe per pair.  Same staging buffer, ordering and waiting rules as the double
 * versions (sfft_run_host_wait drains both kinds). */
int sfft_run_host_f32(sfft_plan *plan, const float *h_R, const float *h_S, float *h_D, double *h_coef);
int sfft_run_host_async_f32(sfft_plan *plan, const float *h_R, const float *h_S, float *h_D, double *h_coef);

/* Per-stage device timing.  sfft_plan_profile(plan, nsteps) with nsteps > 0 makes the next nsteps
 * build/solve/subtract rounds record CUDA events on the plan's stream around each stage (no host
 * synchronisation; 0 disables).  sfft_plan_profile_read synchronises the stream and writes
 * ms[step][SFFT_NUM_STAGES] (row-major; -1 where a stage did not run) for the *nrecorded steps seen.
 * Stage order: 0 row FFT (a1+a2), 1 x-direction lag correlation on the FP64 tensor cores (a3+a4), 2 y-direction
 * pruned inverse DFT to the lag tables (a4), 3 basis-function moments Lambda/Delta (a4'), 4 lag gather (a5),
 * 5 solve (a6), 6 kernel folding + per-row coefficient table (a7), 7 convolve-and-subtract (a7+a8), and the two parts
 * of stage 7 when the subtract takes the Fourier route (-1 on the direct route): 8 FIR along x on the row spectra,
 * 9 inverse row transforms fused with the difference. */
#define SFFT_NUM_STAGES 10
int sfft_plan_profile(sfft_plan *plan, int nsteps);
int sfft_plan_profile_read(sfft_plan *plan, double *ms, int *nrecorded);

/* Number of kernels the plan launched since creation (for bench accounting). */
long sfft_plan_launch_count(const sfft_plan *plan);

void sfft_plan_destroy(sfft_plan *plan);

const char *sfft_strerror(int status);
const char *sfft_last_cuda_error(const sfft_plan *plan);
const char *sfft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SFFT_H_ */
