/*
 * nmf.h -- C-ABI boundary of the B200-native weighted-NMF hot path of
 * arXiv 2309.04623 ("NMF-based GPU accelerated coronagraphy pipeline").
 *
 * The library implements, as hand-written sm_100a CUDA kernels, exactly the
 * steps SURVEY.md section 8(a) lists: component construction by the weighted
 * multiplicative updates of the paper's Eq. 3 (section 2),
 * non-negative projection of science frames on the fixed components
 * ("target modelling") and PSF subtraction.
 *
 * Notation (BASELINE.json orientation; the paper writes V for Omega):
 *   X      [N,P]  reference library, N frames x P pixels, >= 0 where Omega > 0
 *   Omega  [N,P]  weights; 0 = occulted / bad pixel ("missing data"),
 *                 else inverse variance (Eq. 2)
 *   W      [N,K]  coefficients            H [K,P] components
 * Everything is fp32, row-major, innermost index contiguous.
 *
 * General rules for every entry point
 *   - Pointers named *_dev / documented "device" are CUDA device pointers owned
 *     by the caller (e.g. torch tensors); pointers documented "host" are plain
 *     host memory.  The library never frees or keeps a user pointer after the
 *     call's work has been enqueued, except the workspace set on the plan.
 *   - Device base pointers must be 16-byte aligned and P % 4 == 0
 *     (128-bit / TMA loads).  Violations return NMF_ERR_ALIGNMENT.
 *   - Calls are asynchronous: they enqueue work on the plan's stream and return
 *     without synchronising, unless stated otherwise (nmf_objective,
 *     nmf_*_host).  The plan's workspace is used by every call, so calls on one
 *     plan must be stream-ordered (one stream per plan).
 *   - Return value: NMF_OK (0) or a negative nmf_status code.  No exceptions and
 *     no abort cross this boundary.  Asynchronous CUDA faults surface at the next
 *     call or at nmf_objective / a *_host call.
 *   - Numerical conventions: entries with Omega == 0 are
 *     skipped (select semantics; X may hold NaN/Inf there); every ratio is
 *     num / max(den, 1e-30f); H is updated first, then W with the new H.
 *   - Preconditions that are documented, not checked: X >= 0 and finite where
 *     Omega > 0; Omega >= 0; W, H, coef >= 0 on entry (an exact zero stays zero).
 *   - Results are bitwise reproducible run to run for a fixed plan shape on a
 *     fixed device (all cross-CTA sums are fixed-order).
 *   - Arithmetic.  Inputs and results are fp32.  The default (tensor-core) kernel
 *     families evaluate the six contractions of Eq. 3 with every fp32 operand split
 *     exactly into three BF16 pieces and six piece products per product, accumulated
 *     in fp32 (dropped terms <= 2^-22 relative, the level of a 3xTF32 split); the
 *     H update divides with the fast reciprocal (<= 2 ulp); sums across CTAs are
 *     fp64 in a fixed order.  The FFMA families (variants 1, 2, 5, 6) use plain fp32 FMA.
 *     Families therefore agree to fp32 rounding level, not bitwise.
 *   - A plan is bound to the CUDA device that was current when it was created;
 *     every call must be made with that device current (else INVALID_ARG).
 */
#ifndef PAPER_2309_04623_NMF_H
#define PAPER_2309_04623_NMF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum nmf_status {
    NMF_OK = 0,
    NMF_ERR_INVALID_ARG = -1, /* null pointer; N/P/K/M/iters out of range; M > max_targets   */
    NMF_ERR_ALIGNMENT   = -2, /* base pointer not 16-byte aligned or P % 4 != 0              */
    NMF_ERR_UNSUPPORTED = -3, /* N > 256, K > 128 or max_targets > 4096 (compiled limits); a
                                 forced variant (2 .. 6) whose kernels do not cover the shape */
    NMF_ERR_WORKSPACE   = -4, /* workspace missing or smaller than nmf_plan_workspace_bytes  */
    NMF_ERR_ARCH        = -5, /* current device is not compute capability 10.x               */
    NMF_ERR_CUDA        = -6, /* CUDA runtime / launch error (sticky until the plan is freed) */
    NMF_ERR_STATIC_LIMIT = -7 /* nmf_objective_static: P > NMF_STATIC_MAX_P (its scratch has a
                                 fixed size)                                                  */
} nmf_status;

#define NMF_MAX_N 256
#define NMF_MAX_K 128
#define NMF_STATIC_MAX_P 4194304LL /* 2048 x 2048 pixels: the limit of nmf_objective_static */

typedef struct nmf_plan nmf_plan; /* opaque; owns host-side launch state only */

/* Create a plan for problems of shape (N frames, P pixels, K components).
 *   batch        >= 1  number of independent problems nmf_fit_batched handles
 *   max_targets  >= 0  largest M accepted by nmf_project / nmf_subtract
 * Binds to the CUDA device that is current at the time of the call.
 * Errors: INVALID_ARG, ALIGNMENT (P % 4), UNSUPPORTED, ARCH, CUDA.            */
int nmf_plan_create(nmf_plan** out, int N, long long P, int K, int batch, int max_targets);

/* Bytes of device scratch the plan needs (split-K partial slabs, objective
 * partials; for K <= 8 also tile-major copies of X and Omega for the streaming
 * kernel: 8 * N * P bytes per problem of the batch).  The caller allocates it (16-byte aligned) and hands it over with
 * nmf_plan_set_workspace; it must stay valid until the plan is destroyed or a
 * new workspace is set.  Contents need no initialisation.                      */
size_t nmf_plan_workspace_bytes(const nmf_plan* plan);
int nmf_plan_set_workspace(nmf_plan* plan, void* workspace_dev, size_t bytes);

/* cudaStream_t to enqueue on, passed as void*.  NULL = the legacy default stream. */
int nmf_plan_set_stream(nmf_plan* plan, void* cuda_stream);

/* Select the kernel family of nmf_fit / nmf_fit_batched / nmf_project:
 *   0  automatic: the fastest family that covers the shape: the split tensor-core
 *      kernels (4) whenever K <= 128 and the operands fit shared memory, else the
 *      fused tensor-core kernel (3), else FFMA (2, 1); launch-bound problems of at most
 *      64 pixel tiles (128 px) in all run the fused FFMA kernel (2); K <= 8 runs the
 *      streaming FP32 kernel (5); a single problem that stays on chip runs the
 *      resident kernel (6)
 *   1  generic two-kernel FFMA path (any N <= 256, K <= 128; also what
 *      nmf_project runs when omega == NULL)
 *   2  fused FFMA per-pixel-tile kernel (K <= 50)
 *   3  fused tcgen05 kernel: one kernel per iteration does both half-steps (K <= 64)
 *   4  split tcgen05 kernels: H half-step kernel + W half-step kernel (K <= 128;
 *      N = 256 only up to K = 96)
 *   5  streaming FP32 kernel: one kernel per iteration, X and Omega cross HBM once,
 *      plain fp32 FMA, no BF16 split (K <= 8; fit only -- nmf_project of such a plan
 *      runs family 4's projection kernel)
 *   6  resident kernel: ALL iterations of a call in one cooperative launch, X, Omega
 *      in shared memory and H in registers throughout, one grid-wide barrier per
 *      iteration (K <= 8, N <= 64, P <= 128 x number of SMs, batch == 1; fit only)
 * A forced family (2 .. 6) that does not cover the plan's shape makes the fit
 * return UNSUPPORTED.  All families compute the updates of Eq. 3; see "Arithmetic"
 * above for how they differ.  Errors: INVALID_ARG (variant outside 0..6).          */
int nmf_plan_set_variant(nmf_plan* plan, int variant);
/* Which family (1..6) nmf_fit will run for this plan.                              */
int nmf_plan_get_variant(const nmf_plan* plan);

int nmf_plan_destroy(nmf_plan* plan); /* frees host state and any internal staging buffers */

/* Component construction: `iters` times { H half-step ; W half-step } of Eq. 3
 * (PAPER.md:48-50), fixed count, no early stop.
 *   X, Omega  device [N,P]   read-only
 *   W         device [N,K]   in: initial coefficients, out: result (in place)
 *   H         device [K,P]   in: initial components,   out: result (in place)
 * Errors: INVALID_ARG (null, iters < 0), ALIGNMENT, WORKSPACE, CUDA.              */
int nmf_fit(nmf_plan* plan, const float* X, const float* Omega, float* W, float* H, int iters);

/* The same for `batch` independent problems of identical shape, stored
 * contiguously: X, Omega [B,N,P]; W [B,N,K]; H [B,K,P].  One launch sequence.     */
int nmf_fit_batched(nmf_plan* plan, const float* X, const float* Omega, float* W, float* H,
                    int iters);

/* Target modelling: non-negative projection of M science frames on fixed H by
 * `iters` W-type updates of Eq. 3, c <- c o (omega o t)H^T / (omega o (cH))H^T,
 * each frame independently.  Runs the plan's tensor-core family when
 * omega is given, the generic FFMA path when omega == NULL.
 *   H       device [K,P]  read-only     target device [M,P] read-only
 *   omega   device [M,P]  read-only, or NULL = all ones
 *   coef    device [M,K]  in: initial coefficients, out: result (in place)
 * Errors: INVALID_ARG (M < 1, M > max_targets, ...), ALIGNMENT, WORKSPACE, CUDA.   */
int nmf_project(nmf_plan* plan, const float* H, const float* target, const float* omega,
                float* coef, int M, int iters);

/* PSF subtraction: out[m,p] = target[m,p] - factor[m] * sum_k coef[m,k] H[k,p]
 * (PAPER.md:89, 99).  Where omega is given and omega[m,p] == 0 the output is
 * `fill` and target[m,p] is not read into the result.
 *   factor  device [M] or NULL = 1 (slot for best-factor finding)
 *   out     device [M,P], may not alias the inputs.                                */
int nmf_subtract(nmf_plan* plan, const float* H, const float* target, const float* coef,
                 const float* omega, const float* factor, float fill, float* out, int M);

/* Component construction with the paper's stopping rule ("until the
 * change in gradient from one step to the next reaches a set value or the maximum
 * number of iterations is reached"; the quantity is not defined there -- reading
 * G21 in DESIGN.md): the cost f of Eq. 2 is evaluated on the device (fp64, fixed
 * order) at the start and after every `check_every` iterations, and the fit stops
 * at the first check t with |f_(t-check_every) - f_t| < tol * f_(t-check_every),
 * else after max_iters iterations.  tol = 0 never stops early (= nmf_fit).
 *   X, Omega, W, H  device, as for nmf_fit (single problem)
 *   iters_done      host, out: iterations performed
 *   f_last          host, out, nullable: cost at the last check (f_0 if none made)
 * SYNCHRONISES once per check (every `check_every` iterations), not per iteration.
 * Errors: INVALID_ARG (check_every < 1, tol < 0 or NaN, ...), ALIGNMENT, WORKSPACE,
 * CUDA.                                                                            */
int nmf_fit_tol(nmf_plan* plan, const float* X, const float* Omega, float* W, float* H,
                int max_iters, int check_every, double tol, int* iters_done, double* f_last);

/* The cost of Eq. 2, sum over Omega>0 of Omega*(X-WH)^2, accumulated
 * in fp64 on the device in a fixed order.  SYNCHRONISES the plan's stream and
 * writes one double to host memory.                                               */
int nmf_objective(nmf_plan* plan, const float* X, const float* Omega, const float* W,
                  const float* H, double* out_host);

/* The same cost for callers that may not allocate (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): no plan, no workspace, and
 * the call itself performs no cudaMalloc / cudaFree / cudaMallocHost -- its scratch
 * (one fp64 partial sum per block of 128 pixels) is a fixed device array inside the
 * library, 256 KB, held by every GPU that loads the library until the process exits.
 *   X, Omega [N,P], W [N,K], H [K,P]   device, fp32, as for nmf_objective; read only
 *   f_out_dev   device, out: ONE double, written in stream order (no host sync)
 *   stream      cudaStream_t of the CURRENT device (NULL = default stream)
 * Limit: P <= NMF_STATIC_MAX_P (2048^2 pixels), else NMF_ERR_STATIC_LIMIT and nothing
 * is launched; N <= 256, K <= 128 as everywhere (UNSUPPORTED).
 * Asynchronous.  Same kernels and summation order as nmf_objective: the result is
 * bitwise the same.  The scratch is shared by ALL calls on a device and keeps the last
 * call's contents; every element a call reads it has written first, so nothing is
 * cleared -- but two calls that overlap on the GPU (different streams, no ordering
 * between them) RACE on it: order them.  Errors: INVALID_ARG, UNSUPPORTED,
 * STATIC_LIMIT, ARCH, CUDA (not sticky: there is no plan).                          */
int nmf_objective_static(const float* X, const float* Omega, const float* W, const float* H,
                         int N, long long P, int K, double* f_out_dev, void* stream);

/* Device staging of the two *_host calls below.  By default the library allocates
 * it on first use (cudaMalloc, freed by nmf_plan_destroy) -- the one place where
 * it allocates device memory on its own.  A caller who wants to own every device
 * buffer hands over `bytes` >= nmf_plan_staging_bytes(plan, M) (M = largest number
 * of science frames passed to nmf_project_subtract_host; 16-byte aligned; valid
 * until the plan is destroyed or the staging is reset with (NULL, 0)); a *_host call
 * that needs more than a caller-provided buffer holds returns NMF_ERR_WORKSPACE.
 * Errors of set_staging: INVALID_ARG, ALIGNMENT.                                   */
size_t nmf_plan_staging_bytes(const nmf_plan* plan, int M);
int nmf_plan_set_staging(nmf_plan* plan, void* staging_dev, size_t bytes);

/* End-to-end convenience for callers whose data lives in HOST memory: copies
 * X, Omega, W, H host->device into the staging buffer (see above), runs nmf_fit,
 * copies W and H back and
 * SYNCHRONISES.  All four pointers are host pointers (pinned memory makes the
 * copies faster but is not required).  W, H are updated in place.                  */
int nmf_fit_host(nmf_plan* plan, const float* X_host, const float* Omega_host, float* W_host,
                 float* H_host, int iters);

/* Host-memory end-to-end projection + subtraction of M science frames on
 * components already resident on the device (H is a DEVICE pointer, e.g. the
 * result of nmf_fit): copies target/omega/coef in, runs nmf_project and
 * nmf_subtract (factor = 1), copies coef and the residual images back and
 * SYNCHRONISES.  omega_host may be NULL.                                           */
int nmf_project_subtract_host(nmf_plan* plan, const float* H_dev, const float* target_host,
                              const float* omega_host, float* coef_host, float fill,
                              float* out_host, int M, int iters);

/* Closest-frame reference selection ("a percentage of the closest
 * frames ... calculated by minimizing for Euclidean norm"; readings G19/G20 in
 * DESIGN.md).  nmf_ref_distance writes the masked squared Euclidean distances
 *   dist[m,n] = sum over pixels with omega_t[m,p] > 0 and Omega[n,p] > 0 of
 *               (target[m,p] - X[n,p])^2
 * between M target frames and the plan's N library frames (masked entries are
 * skipped and may hold NaN/Inf).  Partial sums are fp32 per pixel
 * range and reduced in fp64 in a fixed order (bitwise reproducible).
 *   target device [M,P]   omega_t device [M,P] or NULL = all valid
 *   X      device [N,P]   Omega   device [N,P] or NULL = all valid
 *   dist   device [M,N]   out (fp32, 16-byte aligned)
 * M is not limited by max_targets.  Errors: INVALID_ARG, ALIGNMENT, WORKSPACE, CUDA. */
int nmf_ref_distance(nmf_plan* plan, const float* target, const float* omega_t, const float* X,
                     const float* Omega, int M, float* dist);

/* For every target m the n_sel (1 <= n_sel <= N) references with the smallest
 * dist[m,:], in ascending order of (distance, frame index) -- the percentage of
 * the library to keep is the caller's choice (the paper gives no formula).
 *   dist device [M,N] read-only     idx device [M,n_sel] out (int32)
 * Errors: INVALID_ARG, CUDA.                                                       */
int nmf_ref_select(nmf_plan* plan, const float* dist, int M, int n_sel, int* idx);

/* Derotate + stack (the subtracted frames "are rotated North-up
 * using their position angles ... then combined"; the paper states no convention:
 * readings G22-G24 in DESIGN.md).  Frame m (an ny x nx image, pixel (y, x) at
 * y*nx + x, ny*nx == the plan's P) is rotated by angle_deg[m] degrees, counter-
 * clockwise with x to the right and y up, about the pixel (ny/2, nx/2): output
 * pixel (y, x) samples the input at
 *   xs = cx + cos(a)(x-cx) + sin(a)(y-cy),  ys = cy - sin(a)(x-cx) + cos(a)(y-cy)
 * by bilinear interpolation (fp64 coordinates, exact at multiples of 90 degrees;
 * neighbours with weight <= 1e-6 ignored).  A sample counts only if all its
 * neighbours are inside the image and have omega > 0 (masked pixels may hold
 * NaN/Inf).  out = mean over the frames with a sample, `fill` where
 * there is none; count (nullable) = number of frames averaged.
 *   resid device [M,P] read-only      omega device [M,P] or NULL = all valid
 *   angle_deg device [M] fp32         out device [P]   count device [P] int32 or NULL
 * M is not limited by max_targets.  Errors: INVALID_ARG (ny*nx != P, ...),
 * ALIGNMENT, CUDA.                                                                 */
int nmf_derotate_stack(nmf_plan* plan, const float* resid, const float* omega,
                       const float* angle_deg, int ny, int nx, float fill, float* out,
                       int* count, int M);

/* Number of kernel launches this plan has enqueued so far (bench bookkeeping).     */
long long nmf_plan_launch_count(const nmf_plan* plan);

const char* nmf_status_string(int code);
/* Text of the last CUDA error recorded on the plan ("" if none).                   */
const char* nmf_plan_last_cuda_error(const nmf_plan* plan);

#ifdef __cplusplus
}
#endif
#endif /* PAPER_2309_04623_NMF_H */
