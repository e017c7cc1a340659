/*
 * linmin.h -- C ABI of liblinmin.so: per-pixel fully constrained linear unmixing on one B200.
 *
 * The operation (citations: /root/reference/PAPER.md line + section/equation):
 *   PAPER.md:48-50 (sec. 2.1, eq. 1)   X = A.S + E, zero-mean Gaussian noise.
 *   PAPER.md:54    (eq. 2)             F = sum_pixels sum_channels (X - A.S)^2, separable per pixel.
 *   PAPER.md:63    (eq. 3)             every mixing coefficient >= 0.
 *   PAPER.md:68    (eq. 4)             the coefficients of a pixel sum to one.
 *   PAPER.md:71-73 (sec. 2.2)          solved by IPLS, a primal-dual interior-point least-squares
 *                                      method; convexity of F suffices for convergence.
 *   PAPER.md:88    (sec. 2.3)          "an estimation of the error on the mixing coefficient is
 *                                      directly provided by the Hessian".
 *   PAPER.md:143, 246, 252             the fit RMS, compared with the noise level.
 *
 * Notation here follows BASELINE.json (the paper writes the transpose): for each of N pixels, a
 * spectrum y (L channels) is fitted by a = argmin ||y - A a||^2 s.t. a >= 0, sum(a) = 1 against ONE
 * shared library A (L x R; column r is endmember r; the paper's S^T).  Outputs per pixel: the
 * minimiser a (R), its first-order standard deviations given the per-channel noise std sigma
 * (reading R3), and the RMS residual sqrt(mean_l (y - A a)_l^2) (reading R8).
 *
 * Layouts (all float32, C order):
 *   A[l*R + r]                       L x R, row-major (channel-major)
 *   Y[p*ldY + l]                     one spectrum = L contiguous floats; ldY >= L elements
 *   sigma                            NULL            -> sigma == 1 (noise amplification factors)
 *                                    stride 0        -> one shared vector sigma[l], l < L
 *                                    stride s >= L   -> per pixel, sigma[p*s + l]
 *   coeffs_out[p*R + r], coeff_sigma_out[p*R + r], resid_out[p]
 *
 * Alignment: float32 alignment (4 bytes) is all that is required of any array.  The fast kernels use 16-byte
 * accesses where the arrays allow it: Y (and per-pixel sigma) 16-byte aligned with ldY (the stride) a multiple of
 * 4, coeffs_out / coeff_sigma_out 16-byte aligned.  Arrays that are not take scalar paths -- at R = 32 a coeffs_out
 * that is not 16-byte aligned sends IPLS through the any-size kernel, several times slower; results are the same
 * minimiser either way (every pixel is finished exactly).
 *
 * Ownership: every pointer is owned by the caller; the library never frees or reallocates caller
 * memory.  Outputs must not alias inputs or each other.  `coeff_sigma_out`, `resid_out`, `sigma`
 * and `opts` may be NULL (output skipped / defaults).  Internal workspace (O(R^2 + L R) bytes) is
 * owned by the linmin_library handle.
 *
 * Device entry points (linmin_unmix, linmin_unmix_lib): every data pointer is a DEVICE pointer on
 * the current CUDA device.  Work is enqueued on opts->stream and the call returns without waiting
 * for it: no stream synchronisation, no host round-trip, no arithmetic of the method on the host
 * (both calls can be captured into a CUDA graph).  Argument errors are returned synchronously;
 * asynchronous CUDA errors surface at the next call or stream synchronisation.
 * Host entry point (linmin_unmix_host): every data pointer is a HOST pointer (pinned memory gives
 * full copy bandwidth); the call stages chunks through the device and returns when outputs are
 * complete.
 *
 * There is no CPU fallback anywhere: without a CUDA device every compute call fails with
 * LINMIN_ERR_CUDA.  No exceptions cross this ABI.  Process-wide state: one staging memory pool per
 * device (created on first use, guarded by a mutex, see linmin_trim_memory); nothing else.  Calls on
 * distinct streams, with the same or with different handles, are thread-safe: a solve call reads the
 * handle and writes only its report fields (launch count, timing events: last caller wins) and its
 * per-stream "last use" events (under a mutex).
 *
 * Defaults that differ from the first draft of this boundary (SURVEY.md 8(b) proposed gap_tol 1e-8,
 * feas_tol 1e-6): gap_tol 1e-7, feas_tol 3e-5 -- the measured optimum of IPLS + exact finish
 * together.  Results do not depend on them: every pixel is finished exactly.
 */
#ifndef LINMIN_H_
#define LINMIN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LINMIN_VERSION 200 /* 0.2.0 */

/* status codes: 0 ok, < 0 error, > 0 warning (results valid) */
#define LINMIN_OK 0
#define LINMIN_ERR_INVALID_ARGUMENT (-1)  /* NULL required pointer, N < 0, L < 1, R < 1, ldY < L, bad stride, struct_size */
#define LINMIN_ERR_UNSUPPORTED_SIZE (-2)  /* R > LINMIN_MAX_R or L > LINMIN_MAX_L */
#define LINMIN_ERR_NOT_IMPLEMENTED (-3)   /* kept for ABI stability: every option of this header is implemented */
#define LINMIN_ERR_CUDA (-4)              /* CUDA runtime failure (including: no device) */
#define LINMIN_ERR_OUT_OF_MEMORY (-5)
#define LINMIN_ERR_LIBRARY_NONFINITE (-6) /* A contains NaN or Inf */
#define LINMIN_ERR_COVARIANCE (-7)        /* the noise covariance is not finite / not positive definite */
#define LINMIN_ERR_STATIC_SCRATCH (-8)    /* linmin_detection_thresholds_static only: R > LINMIN_STATIC_MAX_R, the
                                             library's fixed scratch array has no room for that many endmembers */
#define LINMIN_WARN_RANK_DEFICIENT 1      /* R > L: minimiser may be non-unique (PAPER.md:92 asks R <= L) */

#define LINMIN_MAX_R 256
#define LINMIN_MAX_L 512

/* constraint (sto / slo / pos options of IPLS).  A property of the library handle:
 * linmin_library_create reads it from opts, linmin_unmix_lib requires the same value (or opts == NULL). */
#define LINMIN_CONSTRAINT_SUM_TO_ONE 0        /* eq. 3 + eq. 4: the hot path */
#define LINMIN_CONSTRAINT_SUM_LOWER_THAN_ONE 1 /* a >= 0, sum a <= 1: sum-to-one with a slack (all-zero) endmember,
                                                  added BEFORE the centring; the slack is not returned.  At R = 32
                                                  (L <= 256) the same minimiser is computed without a slack: the
                                                  positivity-only result where its sum is <= 1, else the sum-to-one
                                                  result (the problem is convex: the bound is active there) */
#define LINMIN_CONSTRAINT_POSITIVITY_ONLY 2    /* eq. 3 only (NNLS): no centring, no equality constraint.  gap_tol
                                                  and feas_tol are applied at 1/100 of their value (the projections
                                                  of an uncentred library overstate the scale of the gradients) */

/* weighting (sec. 2.3, eq. 5-6: the renormalised problem).  Also a property of the handle.
 * With a covariance, eq. 2 is solved on the whitened data X' = X.L, S' = S.L (C^-1 = L.L^T); the `sigma`
 * argument of the solve calls is then ignored: coeff_sigma is the projected inverse Hessian of the whitened
 * problem (unit noise) and resid is the RMS of the WHITENED residual, sqrt(r'C^-1 r / L) (about 1 when the
 * model fits to the noise; reading R17). */
#define LINMIN_WEIGHTING_NONE 0               /* unweighted fit; sigma used for propagation only */
#define LINMIN_WEIGHTING_SHARED_COVARIANCE 1  /* opts->cov = L x L covariance matrix (row-major, symmetric pos. def.) */
#define LINMIN_WEIGHTING_SHARED_DIAGONAL 2    /* opts->cov = L per-channel noise standard deviations (C = diag(cov^2)) */

/* per-pixel info word (opts->info_out): flags in bits 0-7, then three counters */
#define LINMIN_INFO_CONVERGED 0x01      /* IPLS met its stopping rule */
#define LINMIN_INFO_MAX_ITER 0x02       /* IPLS stopped at max_iter (the exact finish still ran) */
#define LINMIN_INFO_NONFINITE_INPUT 0x04 /* y has NaN/Inf: all outputs of the pixel are NaN */
#define LINMIN_INFO_CHOL_REGULARISED 0x08 /* a Newton-matrix pivot was clamped */
#define LINMIN_INFO_FINISH_FALLBACK 0x10 /* finish hit its pivot/support cap: result feasible, near-optimal, not certified */
#define LINMIN_INFO_BAD_SIGMA 0x20      /* sigma <= 0 or non-finite: coeff_sigma of the pixel is NaN */
#define LINMIN_INFO_LIBRARY_NONFINITE 0x40 /* linmin_unmix only: A holds NaN/Inf, every output of the call is NaN */
#define LINMIN_INFO_COVARIANCE 0x80     /* linmin_unmix only: opts->cov is not finite / not positive definite, every
                                           output of the call is NaN */
#define LINMIN_INFO_ITERATIONS(w) (((w) >> 8) & 0xff)  /* IPLS Newton iterations */
#define LINMIN_INFO_PIVOTS(w) (((w) >> 16) & 0xff)     /* finish support changes */
#define LINMIN_INFO_SUPPORT(w) (((w) >> 24) & 0xff)    /* number of non-zero coefficients */

typedef struct linmin_opts {
    uint32_t struct_size;       /* sizeof(linmin_opts); anything else -> LINMIN_ERR_INVALID_ARGUMENT */
    void *stream;               /* cudaStream_t; NULL = default stream */
    int64_t ldY;                /* elements between consecutive spectra in Y; 0 -> L */
    int64_t sigma_pixel_stride; /* 0 -> shared sigma[L]; else elements between pixels (>= L) */
    int32_t constraint;         /* LINMIN_CONSTRAINT_* */
    int32_t weighting;          /* LINMIN_WEIGHTING_* */
    int32_t max_iter;           /* IPLS iteration cap, 1..255; 0 -> 50 */
    float gap_tol;              /* stop when a'lambda <= gap_tol * scale; 0 -> 1e-7 */
    float feas_tol;             /* ... and dual/primal residuals <= feas_tol (* scale); 0 -> 3e-5 */
    int32_t *info_out;          /* optional int32[N] (device pointer; host pointer for linmin_unmix_host) */
    int32_t deterministic;      /* results never depend on tiling or scheduling; kept for ABI, always on */
    int32_t reserved;
    const float *cov;           /* weighting != NONE: the shared noise covariance (device pointer; host pointer for
                                   linmin_unmix_host); read by linmin_library_create / linmin_unmix only */
} linmin_opts;

typedef struct linmin_library linmin_library; /* opaque: precomputed per-library data on the device */

/* Once-per-library precompute ("S.S^T"): centred library, Gram
 * matrices in fp32 and fp64, and the start-point data of IPLS (inverse of the regularised Gram
 * matrix) -- all computed by kernels on opts->stream.  A is a DEVICE pointer (copied; the caller may
 * free it afterwards).  Synchronises the stream ONCE, at the end, to read the device flag that says
 * whether A is finite.  Returns LINMIN_OK, LINMIN_WARN_RANK_DEFICIENT (handle valid) or an error
 * (*lib = NULL; LINMIN_ERR_LIBRARY_NONFINITE for NaN/Inf in A, LINMIN_ERR_COVARIANCE for a covariance that is not
 * positive definite).  opts->stream, constraint, weighting and cov are read. */
int linmin_library_create(const float *A, int32_t L, int32_t R, const linmin_opts *opts,
                          linmin_library **lib);

/* Frees the handle's device memory, stream-ordered on the creation stream AFTER the last work enqueued
 * with the handle on any stream (the library records an event per stream it served and the creation
 * stream waits for them).  Exception: work captured into a CUDA graph is not tracked -- keep the handle
 * alive as long as the graph may be launched.  NULL is a no-op. */
void linmin_library_destroy(linmin_library *lib);

/* Unmix N spectra against a precomputed library.  Device pointers on the handle's device (another
 * current device -> LINMIN_ERR_INVALID_ARGUMENT).  N == 0 is a no-op; N >= 2^32 ->
 * LINMIN_ERR_UNSUPPORTED_SIZE.  Enqueues and returns. */
int linmin_unmix_lib(const linmin_library *lib, const float *Y, const float *sigma, int64_t N,
                     const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out,
                     float *resid_out);

/* One-shot form: precompute + solve + release, all enqueued on opts->stream; returns without waiting.
 * Device pointers.  Since nothing is read back, a non-finite library and a covariance that is not positive
 * definite are reported through the OUTPUTS: all of them NaN, every info word = LINMIN_INFO_LIBRARY_NONFINITE
 * and / or LINMIN_INFO_COVARIANCE (linmin_library_create reports them as a status instead:
 * LINMIN_ERR_LIBRARY_NONFINITE, LINMIN_ERR_COVARIANCE).
 * Cost: every call repeats the once-per-library precompute, part of which runs on ONE thread block (start-point data,
 * O(R^3); with a covariance its Cholesky factor and inverse, O(L^3): a few milliseconds at L = 512).  For more
 * than one cube against the same library use linmin_library_create + linmin_unmix_lib. */
int linmin_unmix(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L, int32_t R,
                 const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out, float *resid_out);

/* Same operation with HOST buffers (A, Y, sigma, outputs, opts->info_out): chunks of pixels are
 * copied host->device, solved and copied back on alternating streams so that copies overlap the
 * kernels.  Blocks until the outputs are complete.  opts->stream is ignored. */
int linmin_unmix_host(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L,
                      int32_t R, const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out,
                      float *resid_out);

/* Number of kernel launches the last linmin_unmix_lib call on this handle enqueued (for reports). */
int linmin_library_last_launches(const linmin_library *lib);

/* Per-kernel timing for reports (bench.py's roofline): when enabled, linmin_unmix_lib brackets each
 * of its kernels with CUDA events on the call's stream.  linmin_library_last_timing blocks until the
 * last call's events have completed and returns the device time of the projection+IPLS kernel and of
 * the finish/uncertainty/residual kernel in milliseconds.  The two always add up to the whole call; with
 * sum-lower-than-one at R = 32 (two passes, see LINMIN_CONSTRAINT_SUM_LOWER_THAN_ONE) ipls_ms holds the whitening,
 * the whole positivity-only pass and the IPLS kernels of the sum-to-one pass, finish_ms the sum-to-one finish and
 * the per-pixel selection.  Returns LINMIN_ERR_INVALID_ARGUMENT when timing is disabled or no call was made.
 * Not thread-safe per handle. */
int linmin_library_enable_timing(linmin_library *lib, int enable);
int linmin_library_last_timing(const linmin_library *lib, float *ipls_ms, float *finish_ms);

/* Staging memory (per-call workspaces of linmin_unmix_lib, the device buffers of linmin_unmix_host) is taken
 * from a memory pool the library owns, one per device, and kept between calls.  linmin_trim_memory() returns
 * what is not in use to the driver (call it when idle; the next call allocates again).  Thread-safe. */
int linmin_trim_memory(void);

/* ---------------------------------------------------------------------------------------------------------
 * NEXT rows 3-4 of SURVEY.md 8(f): library builder, detection layer, autofit.  Device pointers; `stream` is a
 * cudaStream_t (NULL = default stream); all enqueue and return unless stated otherwise.
 */

/* The paper's additional spectra: n_extra = 4 -> Flat 1, Flat 0.0001, Slope increasing,
 * Slope decreasing; n_extra = 12 -> also cos, sin, -cos, -sin over a quarter period and over half a period of the
 * spectral domain (reading R18).  Written as columns col0 .. col0 + n_extra - 1 of the L x ld_out
 * row-major library `out`; wavelength: L increasing values (position = normalised wavelength) or NULL (position =
 * l / (L - 1)). */
int linmin_additional_spectra(const float *wavelength, int32_t L, int32_t n_extra, float *out, int32_t ld_out,
                              int32_t col0, void *stream);

/* Detection threshold per endmember, eq. 8, from a LABELLED set: coeffs N x R estimated
 * coefficients, present N x R bytes (non-zero: the endmember is part of the true mixture).  A+ / A- are the
 * detections (coefficient > 0) on present / absent pixels; population std; an empty class contributes 0 (R19).
 * thresholds_out: R floats.  Sums in fp64 in a fixed order (results do not depend on scheduling). */
int linmin_detection_thresholds(const float *coeffs, const unsigned char *present, int64_t N, int32_t R,
                                float *thresholds_out, void *stream);

/* The same with the class definition as an argument.  whole_class = 0: as above (reading R19: A+ / A- are the
 * detections, estimate > 0 -- the green / red points of the paper's Fig. 4).  whole_class = 1: every pixel of each
 * class enters the mean and the std, estimates of exactly 0 included -- PAPER.md:131 defines the classes by the TRUE
 * coefficient ("~30 ... non-null ... A^positive", "~970 ... null ... A^false"), and the paper's interior-point
 * iterate never returns an exact 0, so this is what its eq. 8 ran over; here the exact finish returns exact zeros
 * for most absent endmembers and the two readings differ (R19 has the measured size). */
int linmin_detection_thresholds_ex(const float *coeffs, const unsigned char *present, int64_t N, int32_t R,
                                   int32_t whole_class, float *thresholds_out, void *stream);

/* The thresholds of linmin_detection_thresholds (whole_class = 0) for callers that cannot let the library allocate device memory: an application that gave the
 * whole GPU to its own arena at start-up (an allocation made here would fail or take memory it has planned for),
 * or a latency-bound loop that cannot afford the device-wide synchronisation and unbounded duration an allocation
 * may cost.  linmin_detection_thresholds draws its per-block partial sums from the library's staging pool; this
 * call keeps them in ONE fixed array inside the library image and calls no cudaMalloc / cudaFree, no pool and no
 * other allocating routine.  Inputs and outputs are the caller's, as above.
 *   Limit: R <= LINMIN_STATIC_MAX_R (else LINMIN_ERR_STATIC_SCRATCH; nothing is launched); N is not limited (at most
 *     LINMIN_STATIC_MAX_BLOCKS thread blocks walk the data).  The array takes LINMIN_STATIC_MAX_BLOCKS x
 *     LINMIN_STATIC_MAX_R x 6 doubles = 384 KiB on every GPU that loads the library, until the process exits.
 *   First call on a device: looks the array's address on that device up (once, kept afterwards).  Make that first
 *     call during set-up, before any stream capture is begun.
 *   Sharing: every call on a device uses the same array, which still holds the previous call's sums.  Nothing has
 *     to be cleared (each call overwrites every slot it later reads), but two calls that overlap on the GPU -- on two
 *     streams, or from two host threads -- race on it and return garbage: keep calls on one device in stream order.
 *   Result: the blocks' fp64 sums are added in a fixed order, but the launch has fewer blocks than the pooled
 *     call's, so the float32 thresholds equal linmin_detection_thresholds' to rounding (1 ulp), not always bit for
 *     bit; repeated calls on the same data return the same bits. */
#define LINMIN_STATIC_MAX_R 64
#define LINMIN_STATIC_MAX_BLOCKS 128
int linmin_detection_thresholds_static(const float *coeffs, const unsigned char *present, int64_t N, int32_t R,
                                       float *thresholds_out, void *stream);

/* The three detection conditions of PAPER.md:239-246: mask[p*R + i] = coeffs > thresholds[i] and coeff_sigma < coeffs
 * and resid[p] < rms_max ("10 times the dark current noise").  counts_out (optional): R detections per endmember. */
int linmin_detect(const float *coeffs, const float *coeff_sigma, const float *resid, const float *thresholds,
                  float rms_max, int64_t N, int32_t R, unsigned char *mask_out, unsigned long long *counts_out,
                  void *stream);

/* Second pass "with the detected spectrum only": linmin_unmix against the columns of A whose byte in
 * keep (R bytes, device) is non-zero; coefficients and uncertainties of the other endmembers are 0.  SYNCHRONISES
 * opts->stream TWICE: once to read `keep` (the size of the sub-library decides the allocations) and once after
 * uploading the column list (a host array that does not outlive the call).  Not capturable into a CUDA graph. */
int linmin_second_pass(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L, int32_t R,
                       const unsigned char *keep, const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out,
                       float *resid_out);

/* "Autofit" degeneracy test of a library (eq. 7): for every endmember n the residue E of its best
 * fit by all the OTHER endmembers, unconstrained (resid_ls_out, L x R, column n) and under positivity
 * (resid_nn_out, L x R; the pos option of the solver).  Either output may be NULL. */
int linmin_autofit(const float *A, int32_t L, int32_t R, void *stream, float *resid_ls_out, float *resid_nn_out);

const char *linmin_strerror(int code);
int linmin_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LINMIN_H_ */
