/* sfft.h -- C ABI of libsfft.so: B200 (sm_100a) SFFT image differencing of one aligned
 * reference/science CCD pair.
 *
 * Method: PAPER.md:40 (§1) "formulates the image subtraction problem in the Fourier domain and
 * accounts for spatial variations in the point-spread function ... convolution kernel is
 * modeled with a delta-function basis"; used once per science image (§2.3.2).
 * The paper prints no equations; BASELINE.json `north_star` fixes the problem, SURVEY.md §8.0
 * and DESIGN.md ("Readings") fix every convention used below:
 *
 *   D = S - ( R (x) K(x,y) + B(x,y) ),  circular convolution on the H x W grid,
 *   xi(x) = (2x+1-W)/W, eta(y) = (2y+1-H)/H, monomials P_t = xi^p eta^q ordered
 *     for d in 0..D: for q in 0..d: p = d-q,
 *   shifts s <-> (u,v), u,v in [-w,w], s = (v+w)(2w+1)+(u+w), u along x (fastest axis),
 *   model  M(x,y) = sum_t sum_s a[s,t] (P_t R)((x-u) mod W,(y-v) mod H) + sum_t' beta[t'] P_t'(x,y)
 *   coefficient vector c (length N = (2w+1)^2 (DK+1)(DK+2)/2 + (DB+1)(DB+2)/2):
 *     c[t*L + s] = a[s,t]  (L = (2w+1)^2),  c[L*T_K + t'] = beta[t'],
 *   fit: good-pixel indicator m = (mask==0); R~_t = m P_t R, S~ = m S, Psi_t' = m P_t';
 *     A = G^T G, b = G^T S~ with G's columns the shifted R~_t and the Psi_t'  (normal equations,
 *     no weights, no regularisation); c = A^-1 b by Cholesky.
 *
 * Memory: every image/matrix pointer below is a DEVICE pointer owned by the caller, 16-byte
 * aligned, contiguous; images are H rows x W columns, row-major, element (y,x) at y*W+x, fp64.
 * The library never allocates, frees or modifies caller buffers other than the stated outputs.
 * The four hot calls only enqueue work on `stream` (a cudaStream_t passed as void*; NULL = the
 * legacy default stream): they never synchronise the stream or the device.  Internally a plan also
 * owns one side stream that is forked from and joined back into `stream` with events inside a call
 * (or between sfft_subtract_prepare and the sfft_subtract that consumes it); the caller never sees it.
 * A plan owns scratch memory and is NOT re-entrant: use one plan per stream in flight.  No call throws; every call
 * returns an sfft_status.  There is no CPU fallback: without a CUDA device plan creation fails.
 */
#ifndef SFFT_H
#define SFFT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sfft_plan sfft_plan; /* opaque; owns workspace, twiddle and index tables */

typedef enum {
  SFFT_OK = 0,
  SFFT_ERR_INVALID_ARG = 1, /* NULL where not allowed, misaligned pointer, bad sizes */
  SFFT_ERR_UNSUPPORTED = 2, /* size/degree outside what this build supports */
  SFFT_ERR_ALLOC = 3,       /* cudaMalloc / host allocation failed */
  SFFT_ERR_CUDA = 4         /* a CUDA runtime call or launch failed (incl. no device) */
} sfft_status;

/* Create a plan for H x W images, kernel half-width w, polynomial degrees DK (kernel) and DB
 * (background).  Supported: H, W powers of two, 16 <= H, W <= 4096; 0 <= w <= 15, 4w+1 <= min(H,W);
 * 0 <= DK, DB <= 3.  Otherwise SFFT_ERR_UNSUPPORTED.  w <= 5 (every BASELINE configuration) runs the tuned
 * kernels; w > 5 (lag half-ranges above 10) runs the generic column/cross kernels with the lag range split
 * into windows and a plain mixing kernel -- same results, not tuned.  Allocates scratch on the current
 * device (it grows with N^2: N = 9620 for w = 15, DK = 3) and uploads tables; may synchronise.  *out is set
 * to NULL on failure.
 * (north_star: sfft_plan_create(H,W,w,DK,DB).) */
sfft_status sfft_plan_create(sfft_plan** out, int H, int W, int w, int DK, int DB);

/* Free a plan and its scratch.  The caller must have synchronised every stream that used it. */
sfft_status sfft_plan_destroy(sfft_plan* p);

/* N, the number of unknowns (length of b and coeffs, order of A).  -1 if p is NULL. */
int sfft_num_coeffs(const sfft_plan* p);

/* Bytes of device scratch the plan owns (0 if p is NULL). */
size_t sfft_workspace_bytes(const sfft_plan* p);

/* Static, human-readable name of a status code. */
const char* sfft_status_string(sfft_status s);

/* Build the normal equations (north_star subsystems (1)-(4)):
 * weighted masked images -> batched fp64 2-D real FFTs -> Fourier-domain cross products and
 * inverse transforms restricted to the lag window -> gather into A and b.
 *   R, S  in : H*W fp64 (device).      mask in: H*W uint8 (device, 16-byte aligned), nonzero = excluded; NULL = none.
 *   A    out : N*N fp64 row-major, FULL symmetric matrix (both triangles written).
 *   b    out : N fp64.
 * Errors: INVALID_ARG on NULL p/R/S/A/b or misalignment; CUDA on a launch failure. */
sfft_status sfft_build_system(sfft_plan* p, const double* R, const double* S,
                              const unsigned char* mask, double* A, double* b, void* stream);

/* The same system for the LITERAL objective "minimise sum D^2 over unmasked pixels" (north_star;
 * SURVEY.md §8(f) NEXT-1): R and S are used as they are and the masked pixels are dropped from the
 * sum, A = sum_{x unmasked} g(x) g(x)^T, b = sum_{x unmasked} g(x) S(x), g(x) the design-matrix row of
 * the unmasked images.  Computed as sfft_build_system with mask = NULL minus the masked pixels'
 * rank-one terms: fully masked rows and columns (a CCD's border frame; up to 32 per direction) through
 * 1-D correlations of a few image rows / columns, every other masked pixel through a symmetric rank-K
 * update (~0.4 ms more than the ordinary build at the full CCD with a 6-pixel border, + ~40 ns per
 * isolated masked pixel).  Recovers a known kernel exactly under any mask, which the input-masking
 * system of sfft_build_system cannot (reading A2').  Same arguments and errors, plus
 * SFFT_ERR_UNSUPPORTED (nothing enqueued) when mask != NULL and N > 2047, which only kernel half-widths
 * w > 5 can reach (the rank-K update keeps the whole triangle of A in one cooperative launch); for w > 5
 * every masked pixel takes the rank-K update (the line shortcut is compiled for w <= 5). */
sfft_status sfft_build_system_exact(sfft_plan* p, const double* R, const double* S,
                                    const unsigned char* mask, double* A, double* b, void* stream);

/* Solve A c = b by blocked fp64 Cholesky + two triangular solves (north_star (5), a5).
 *   A, b in (device, not modified; only the lower triangle of A is read), coeffs out: N fp64.
 *   info out (device int, may be NULL): 0 = ok; k > 0 = the leading minor of order k is not
 *   positive (A not positive definite; coeffs are then unspecified).  Reported on the device so
 *   the stream is never stalled. */
sfft_status sfft_solve(sfft_plan* p, const double* A, const double* b, double* coeffs,
                       int* info, void* stream);

/* Apply the fitted spatially varying kernel and background and subtract (north_star (6), a6):
 * D = S - M, on EVERY pixel from the raw (unmasked) R and S.
 *   R, S in: H*W fp64; coeffs in: N fp64 (device); D out: H*W fp64, must not alias R or S. */
sfft_status sfft_subtract(sfft_plan* p, const double* R, const double* S, const double* coeffs,
                          double* D, void* stream);

/* Optional overlap hint.  The first stage of sfft_subtract (row transforms of xi^p R) does not need
 * the coefficients: this call enqueues it on the plan's side stream, ordered after everything already
 * enqueued on `stream` and concurrent with what the caller enqueues next -- typically sfft_solve,
 * which is latency-bound and leaves most SMs idle.  The next sfft_subtract on this plan with the SAME
 * R pointer waits for it and skips that stage; any other R, or an intervening sfft_build_system,
 * discards the prepared data.  Contract: R is not modified between this call and that sfft_subtract.
 * Results are bitwise those of sfft_subtract alone.  Call order: build_system, subtract_prepare,
 * solve, subtract. */
sfft_status sfft_subtract_prepare(sfft_plan* p, const double* R, void* stream);

/* ---- steps that follow the differencing of one CCD ---------- */

#define SFFT_MAX_TEMPLATES 9

/* Multi-template combination (§2.3.2: the N_TEMP difference images of one science
 * exposure are "normalized to a common photometric zero point ... and median-combined"; N_TEMP
 * defaults to 5):  out[i] = median over k of scale[k] * D[k][i],  i < npix.
 * For even n the median is the mean of the two middle values (reading M1); a NaN in any of
 * the n values makes out[i] NaN (reading M2).
 *   D     in : HOST array of n DEVICE pointers, each npix fp64, 16-byte aligned, none aliasing out.
 *   scale in : HOST array of n flux factors (10^(0.4 (zp_ref - zp_k))).
 *   out  out : npix fp64 (device, 16-byte aligned).      1 <= n <= SFFT_MAX_TEMPLATES.
 * Enqueues one kernel on `stream`; never synchronises.  Needs no plan. */
sfft_status sfft_median_combine(const double* const* D, const double* scale, int n, size_t npix,
                                double* out, void* stream);

/* Multi-template MODE (§2.3.2: "the science image is differenced against each individual
 * template exposure, producing N_TEMP difference images per science exposure.  All difference images
 * are subsequently normalized to a common photometric zero point ... and median-combined"; N_TEMP
 * default 5).  One call = n x (sfft_build_system, sfft_solve, sfft_subtract) against the
 * same science image S, then sfft_median_combine.  The science image's share of the build -- the row
 * transform of m S and its row moments -- is computed for the first template only and reused by the
 * other n - 1 builds, which is why ONE mask serves all n fits (reading MT1: the union of the
 * science and template data-quality masks; NULL = none).  Every D_k, c_k is bitwise what the three
 * separate calls give for (R[k], S, mask).
 *   R      in : HOST array of n DEVICE pointers, each H*W fp64, 16-byte aligned.
 *   scale  in : HOST array of n flux factors to the common zero point.
 *   Dk    out : n*H*W fp64 (device): the individual difference images D_k (unscaled).
 *   coeffs out: n*N fp64 (device);  info out (nullable): n ints (device), as sfft_solve.
 *   out   out : H*W fp64 (device): median_k(scale[k] * D_k).    1 <= n <= SFFT_MAX_TEMPLATES.
 * All work is enqueued on `stream` (and the plan's side stream, joined back); never synchronises. */
sfft_status sfft_multi_template_difference(sfft_plan* p, const double* const* R, const double* S,
                                           const unsigned char* mask, const double* scale, int n,
                                           double* Dk, double* coeffs, int* info, double* out, void* stream);

/* The same mode with the n chains spread over several plans (the GPU works
 * through a queue of independent differencings): template k runs on plans[k % nplans], so the
 * latency-bound sfft_solve of one template overlaps the transforms of the others.  plans[0]'s chains are
 * enqueued on `stream`; every other plan's go to a stream that plan owns, forked from `stream` at entry
 * and joined back into it before the median (also on every error return) -- no host synchronisation,
 * and work enqueued on `stream` after the call sees all outputs.  Each plan transforms m S once (for
 * its first template).  Results are bitwise those of sfft_multi_template_difference.
 *   plans in : HOST array of nplans distinct plans created with the same (H, W, w, DK, DB), none in
 *              use by other in-flight work;  1 <= nplans <= SFFT_MAX_TEMPLATES (plans beyond n are
 *              left untouched).  sfft_plan_set_solve_ctas applies per plan (a cap of about 16 CTAs
 *              lets the solves run beside the other plans' transforms).
 * Other arguments and errors as sfft_multi_template_difference (N, H, W are plans[0]'s). */
sfft_status sfft_multi_template_difference_plans(sfft_plan* const* plans, int nplans, const double* const* R,
                                                 const double* S, const unsigned char* mask, const double* scale,
                                                 int n, double* Dk, double* coeffs, int* info, double* out,
                                                 void* stream);

/* Monte-Carlo limiting flux of a difference image (§2.3.3: "aperture fluxes at 1024
 * randomly selected background positions ... deriving the 5 sigma threshold from their standard
 * deviation").  The positions are INPUTS (the random draw is the caller's).
 *   D in: H*W fp64 (device);  mask in: H*W uint8 (device), nonzero = not background, NULL = none.
 *   xs, ys in: n real-valued pixel positions (device; pixel (y,x) is centred at integer coordinates).
 *   flux out: n fp64 (device): sum of D over the pixels whose centres lie within `radius` of the
 *     position; NaN when that disc leaves the frame or touches a masked pixel, or when the position
 *     itself is not finite (readings L1, L2).
 *   stats out: 3 fp64 (device): number of kept positions, their mean flux, their population
 *     standard deviation sigma.  The limiting magnitude is zp - 2.5 log10(5 sigma) (host arithmetic).
 * 0 < radius <= 64.  Enqueues two kernels on `stream`; never synchronises.  Needs no plan. */
sfft_status sfft_aperture_stats(const double* D, const unsigned char* mask, int H, int W,
                                const double* xs, const double* ys, int n, double radius,
                                double* flux, double* stats, void* stream);

/* Three-channel stamps for the real-bogus classifier (§2.3.4: "three-channel image
 * stamps -- consisting of the science image, template image, and their difference -- centered on the
 * candidate position").  The paper fixes neither the size nor an edge rule; readings ST1-ST4:
 * channel order (science, template, difference); the stamp is size x size pixels and its centre pixel
 * (index size/2 along each axis) is the pixel nearest the position, (floor(x + 1/2), floor(y + 1/2)),
 * pixel (y,x) centred at integer coordinates; pixels outside the frame are 0; a non-finite position
 * gives an all-NaN stamp.
 *   S, R, D in: H*W fp64 (device);  xs, ys in: n real-valued positions (device);
 *   out: n*3*size*size fp64 (device), out[k][channel][j][i].   1 <= size <= 1024.
 * A gather (bit-exact copies).  Enqueues one kernel on `stream`; needs no plan. */
sfft_status sfft_cut_stamps(const double* S, const double* R, const double* D, int H, int W,
                            const double* xs, const double* ys, int n, int size, double* out, void* stream);

/* Resampling onto another pixel grid, the step before the differencing (§2.3.2: the
 * science image is reprojected "onto the WCS of the corresponding template image(s) using SWARP";
 * archival exposures are "resampled onto the expected WCS of the target CCD").  The
 * paper fixes neither the interpolant nor a WCS; readings R1-R4: the pixel map is affine,
 *   x_in = M[0] + M[1] x_out + M[2] y_out,   y_in = M[3] + M[4] x_out + M[5] y_out
 * (pixel centres at integer coordinates; M is a HOST array of 6), the interpolant is the separable
 * Lanczos kernel of order a (1..4; SWarp's default is 3) with the 2a x 2a weights divided by their
 * sum and no Jacobian flux factor; an output pixel whose taps leave the input frame is 0.
 *   in: Hin*Win fp64 (device); out: Hout*Wout fp64 (device, not aliasing in);
 *   outside (nullable): Hout*Wout uint8 (device), 1 where the taps left the frame, else 0.
 * Enqueues one kernel on `stream`; needs no plan. */
sfft_status sfft_resample_affine(const double* in, int Hin, int Win, const double* M, int a, double* out,
                                 int Hout, int Wout, unsigned char* outside, void* stream);

/* The same resampling for a data-quality mask ("the resampled ood images are discretized
 * using an empirical threshold of 0.3: pixels with values above 0.3 are flagged as bad (set to 2^1),
 * and others are flagged as good (set to 2^0)").  in: uint8, nonzero = bad; the 0/1 indicator is
 * interpolated with the weights above; out: 2 where the value exceeds `threshold` or the taps leave
 * the frame, else 1 (reading R5).  To use the result as the `mask` of sfft_build_system map 1 -> 0. */
sfft_status sfft_resample_mask_affine(const unsigned char* in, int Hin, int Win, const double* M, int a,
                                      double threshold, unsigned char* out, int Hout, int Wout,
                                      void* stream);

/* ---- diagnostics (not on the hot path) ------------------------------------------------------ */

/* Per-stage device times of the most recent build/solve/subtract calls are NOT recorded by the
 * hot calls (they never synchronise).  This helper runs a dependent-free DFMA loop on every SM
 * for `iters` iterations on `stream`, synchronises it, and returns the achieved fp64 rate in
 * *tflops: the measured FP64-pipe peak used as the "alu" roofline denominator.
 * kind = 0: DFMA (CUDA-core fp64 pipe); kind = 1: DMMA (mma.sync m8n8k4 f64). */
sfft_status sfft_probe_fp64(int kind, int iters, double* tflops, double* elapsed_ms, void* stream);

/* Optional per-stage timing for benchmarks.  With profiling on, every hot call records a CUDA
 * event pair on the caller stream around each stage (no synchronisation; at most 512 pending
 * pairs between reads).  sfft_profile_read synchronises on the pending events, folds them into
 * per-stage totals and returns the accumulated milliseconds and pair count of `stage`:
 *   0 build: row pass (k_row2_fwd)          1 build: column pass (k_col_fwd), or the fused
 *                                            column/cross kernel (k_colb)
 *   2 build: cross+pruned inverse, K-K     3 build: cross+pruned inverse, K-S
 *   4 build: lag-row inverse + moments + gather      5 solve (all kernels)
 *   6 subtract: row pass   7 subtract: phase table + y-mixing   8 subtract: inverse rows + D
 *   9 build: sparse part of the kernel-background block (special-pixel list + correction sums)
 * reset != 0 clears that stage's totals after reading. */
sfft_status sfft_profile_enable(sfft_plan* p, int on);
sfft_status sfft_profile_read(sfft_plan* p, int stage, double* total_ms, int* count, int reset);

/* Number of kernel launches the last call of each hot entry point enqueued (host-side counter,
 * for bench.py's "gpu_launches"): which = 0 build, 1 solve, 2 subtract.  -1 on bad arguments. */
int sfft_last_launch_count(const sfft_plan* p, int which);

/* 1 if the plan runs the fused (blocked) column/cross-spectra kernel (H in {1024, 2048, 4096} and at
 * most 32 map pairs, i.e. DK <= 2), 0 if it runs the separate column-pass and cross kernels, -1 if
 * p is NULL.  Both are CUDA paths with identical results up to rounding order; profile stage 1 then
 * holds the fused kernel and stages 2, 3 stay empty. */
int sfft_plan_fused(const sfft_plan* p);

/* Throughput knob for pipelines that keep several plans in flight on different streams: caps the
 * number of CTAs of the cooperative Cholesky kernel (default 0 = one per SM, the lowest latency for
 * a single pair).  A smaller grid leaves whole SMs to the other plans' transform kernels while this
 * plan's latency-bound solve runs.  Results are bitwise independent of the setting. */
sfft_status sfft_plan_set_solve_ctas(sfft_plan* p, int max_ctas);

/* sfft_solve for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same Cholesky kernels as sfft_solve (north_star
 * (5), a5), but no plan -- the factorisation workspace is a static array inside the library instead of a
 * plan's cudaMalloc'ed scratch.  The call performs NO cudaMalloc / cudaFree and calls no allocating
 * library routine; it only enqueues work on `stream`.
 *   A    in : N*N fp64 row-major (device, not modified; only the lower triangle is read).
 *   b    in : N fp64 (device, not modified).      coeffs out: N fp64 (device).
 *   info out: device int, may be NULL; meaning as in sfft_solve.
 *   N       : 1 <= N <= SFFT_SOLVE_STATIC_MAX_N (the Full configuration has N = 732).
 * Limit and cost: the static workspace holds (MAX_N + 1) * MAX_N fp64 = 4.7 MB and is resident on every
 * GPU that loads the library, until the process exits.  N > SFFT_SOLVE_STATIC_MAX_N returns
 * SFFT_ERR_UNSUPPORTED (nothing is enqueued); N < 1 or a NULL A/b/coeffs returns SFFT_ERR_INVALID_ARG.
 * Sharing: ALL calls on a device use the one workspace, which keeps the previous call's contents (the
 * call rewrites every word it later reads, and clears its grid-barrier words itself).  Two calls that
 * overlap on the GPU (different streams, or different host threads' streams) RACE and give wrong results:
 * order them on one stream or with events.  Results are bitwise those of sfft_solve. */
#define SFFT_SOLVE_STATIC_MAX_N 768
sfft_status sfft_solve_static(const double* A, const double* b, int N, double* coeffs, int* info,
                              void* stream);

/* Library version string, e.g. "sfft-b200 0.1 (sm_100a)". */
const char* sfft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SFFT_H */
