/*
 * kcs.h -- C ABI of libkcs.so: one ICM iteration of Kinetic Compressive Sensing on one B200 (sm_100a).
 *
 * Citations:  P:<n> = /root/reference/PAPER.md line n (arXiv 1803.10045);  BJ = BASELINE.json;
 *             Qn / P1-P5 / O1-O2 / K1-K6 / L1-L3 / I = the frozen readings listed in DESIGN.md section 3.
 *
 * Conventions
 *   - Every function returns int: 0 = KCS_OK, negative = error (kcs_last_error() gives a message).
 *     No C++ exception crosses this boundary.
 *   - OWNERSHIP: the caller owns every data buffer.  Unless a parameter is marked [host], data
 *     pointers are DEVICE pointers to fp32, C order, x fastest.  The library owns only the opaque
 *     kcs_ctx (geometry tables, per-subset sensitivity, kinetic tables, workspace).
 *   - ASYNCHRONY: every compute call only enqueues work on the context's CUDA stream and returns;
 *     it never synchronises.  (kcs_create / kcs_destroy synchronise that stream.)
 *   - External ("planar") layouts:
 *        activity   x[T][nz][ny][nx]
 *        sinogram   y[T][nz][A][B]            subset sinogram  y_s[T][nz][A/S][B]  (local angle la <-> a = s + la*S)
 *        maps       theta[4][nz][ny][nx]      parameter order (K1, k2, k3, vB)
 *        lambda, cost [nz][ny][nx]
 *     (with kcs_config.n_replicas = N > 1 read N*nz for nz everywhere below)
 *   - Internally the hot path keeps activity and sinograms frame-innermost ([voxel][Tp], Tp = the power
 *     of two >= T, 4..32) so that one cache line fetched for a bilinear tap serves every time frame
 *     (BJ north_star); the pack/unpack transposes are part of the calls below.
 */
#ifndef KCS_H
#define KCS_H

#ifdef __cplusplus
extern "C" {
#endif

#define KCS_OK 0
#define KCS_ERR_NULL (-1)    /* a required pointer is NULL */
#define KCS_ERR_SHAPE (-2)   /* non-positive size, unsupported geometry ratio, bad subset / frame range */
#define KCS_ERR_SUBSET (-3)  /* n_subsets does not divide n_angles */
#define KCS_ERR_FRAMES (-4)  /* n_frames > KCS_MAX_FRAMES or a frame with t_end <= t_start */
#define KCS_ERR_CUDA (-5)    /* a CUDA runtime call failed (message in kcs_last_error) */
#define KCS_ERR_ALLOC (-6)   /* device or host allocation failed */

#define KCS_MAX_FRAMES 32

#define KCS_PRIOR_POISSON_MATCHED 0 /* Q8: sigma^2 = max(F,eps)/S  =>  D = S (1 + beta (x-F)/max(F,1e-20)) */
#define KCS_PRIOR_ABSOLUTE 1        /* literal eq. 3 with an explicit sigma^2: D = S + beta (x-F)/sigma2 */

#define KCS_R_PER_FRAME 0 /* randoms r[T]: one constant per frame */
#define KCS_R_FULL 1      /* randoms r[T][nz][A][B] */

typedef struct kcs_ctx kcs_ctx;

/* Problem description (P:67 system matrix p_vd; BJ configs).  All pointers here are [host]. */
typedef struct {
    int nx, ny, nz;                 /* voxels; slices are independent direct planes (BJ configs[2],[3]) */
    float vx, vy, vz;               /* voxel size, mm (P1) */
    int n_angles, n_bins;           /* theta_a = pi*a/n_angles, a = 0..A-1 (Q1); bin centre s_b = (b-(B-1)/2) bin_mm */
    float bin_mm;
    int n_steps;                    /* samples per ray K, u_k = (k-(K-1)/2) step_mm (Q3) */
    float step_mm;
    int n_subsets;                  /* S, must divide n_angles; subset s = {a : a mod S == s} (P5, Q5) */
    int n_frames;                   /* T <= KCS_MAX_FRAMES */
    const double *t_start_min;      /* [host][T] frame start, minutes (fp64: the kinetic tables are built in fp64) */
    const double *t_end_min;        /* [host][T] frame end, minutes */
    float feng_A[3];                /* BJ configs[0](1): Cp(t) = (A1 t - A2 - A3) e^{-l1 t} + A2 e^{-l2 t} + A3 e^{-l3 t} */
    float feng_lambda[3];
    const unsigned char *mask_host; /* [host][ny][nx] field-of-view mask, NULL = Q2 default disc */
    int n_replicas;                 /* N >= 1 (0 is read as 1): noise realisations of one object reconstructed in one
                                     * batch ("100 noisy realizations").  They share geometry, sensitivity, weight
                                     * table and kinetic tables; every buffer then carries N * nz slices, replica-major
                                     * (slice index = replica * nz + z), e.g. x[T][N*nz][ny][nx].  Replicas never interact:
                                     * the 6-neighbourhood of the Huber prior stops at a replica's first and last slice. */
} kcs_config;

/* Create / destroy.  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 * Requires (|cos| vx + |sin| vy)/bin_mm <= 1.5 and (|sin| vx + |cos| vy)/step_mm <= 1.5 for every angle
 * (so each voxel sees at most 3 bins x 3 steps per angle), else KCS_ERR_SHAPE. */
int kcs_create(kcs_ctx **out, const kcs_config *cfg, void *stream);
int kcs_destroy(kcs_ctx *ctx);
/* Change the stream later calls are enqueued on (e.g. a capturing stream). */
int kcs_set_stream(kcs_ctx *ctx, void *stream);
/* Message of the last error on this context ("" if none); ctx may be NULL (create-time errors). */
const char *kcs_last_error(const kcs_ctx *ctx);
/* Bytes of device workspace the context owns. */
long long kcs_workspace_bytes(const kcs_ctx *ctx);
/* Copy the [ny][nx] field-of-view mask in use to a [host] buffer. */
int kcs_get_mask(const kcs_ctx *ctx, unsigned char *mask_host_out);
/* Count of kernel launches this context has enqueued so far (bench.py's gpu_launches). */
long long kcs_launch_count(const kcs_ctx *ctx);

/* for launch-bound volumes (nz*ny*nx*T <= 4e6: C1, C2) kcs_icm_run / kcs_icm_iteration capture their kernel
 * sequence into a CUDA graph on the first call with a given set of arguments and replay it afterwards (pointers and
 * scalars are baked in, buffer contents are read at replay; results are bit-identical to the direct launches).
 * kcs_use_graphs(ctx, 0) turns this off; kcs_graph_replays counts the replays so far. */
int kcs_use_graphs(kcs_ctx *ctx, int on);
long long kcs_graph_replays(const kcs_ctx *ctx);

/* Optional per-kernel timing for the roofline report.  While enabled, every kernel launch of this
 * context is bracketed by CUDA events on the context's stream.  kcs_profile_read SYNCHRONISES the stream, adds the
 * elapsed milliseconds and launch counts since the previous read into ms[class] / count[class] ([host] arrays of
 * n_classes >= KCS_PROFILE_NCLASS entries, overwritten) and clears the records.  Classes: */
#define KCS_PROFILE_PACK 0     /* planar -> frame-innermost transposes */
#define KCS_PROFILE_UNPACK 1   /* frame-innermost -> planar */
#define KCS_PROFILE_KINETIC 2  /* model-curve evaluator (a1) */
#define KCS_PROFILE_FORWARD 3  /* forward projector + fused Poisson ratio (a3, a4) */
#define KCS_PROFILE_BACK 4     /* gather back-projector + fused OSL update (a5, a6) */
#define KCS_PROFILE_LM 5       /* MAP-LM step (a8-a10) */
#define KCS_PROFILE_OTHER 6    /* sensitivity images, stand-alone OSL update */
#define KCS_PROFILE_NCLASS 7
int kcs_profile_enable(kcs_ctx *ctx, int on);
int kcs_profile_read(kcs_ctx *ctx, double *ms, long long *count, int n_classes);

/* P1-P3, P5 (BJ north_star "ray-driven parallel-beam line integrals with bilinear
 * interpolation"):  y_s[f] = A_s x[f]  for frames f in [f0, f0+nf), all batched in one launch.
 *   (A x)[z,a,b] = step_mm * sum_k bilinear(x[z]; sample(a,b,k)), pixels outside the image are 0.
 * subset = -1: all angles (y_s is then y[T][nz][A][B]).  No scale, no randoms.
 * x: full activity [T][nz][ny][nx]; y_s: full [T][nz][A_s][B]; only frames [f0,f0+nf) are read / written. */
int kcs_forward_project(kcs_ctx *ctx, const float *x, float *y_s, int subset, int f0, int nf);

/* P4: b[f] = A_s^T q_s[f], the exact matrix transpose of kcs_forward_project, computed as a gather
 * (no atomics, run-to-run deterministic).  Overwrites b[f] for f in [f0,f0+nf). */
int kcs_back_project(kcs_ctx *ctx, const float *q_s, float *b, int subset, int f0, int nf);

/* A_s^T 1 for one slice (no scale): sens[ny][nx] (device).  subset = -1: all angles. */
int kcs_sensitivity(kcs_ctx *ctx, int subset, float *sens);

/* eq. 2-3 with readings O2, Q7-Q10, for all T frames:
 *   D = S (1 + beta (x-F)/max(F,1e-20))     [KCS_PRIOR_POISSON_MATCHED]
 *   D = S + beta (x-F)/sigma2               [KCS_PRIOR_ABSOLUTE]
 *   x <- x * bp / max(D, 0.1 S);   x <- 0 where S <= 1e-12 max(S) or outside the mask.
 * x in/out [T][nz][ny][nx]; bp = scale A_s^T q, same shape; sens = scale A_s^T 1, [ny][nx]; F same shape as x. */
int kcs_osl_update(kcs_ctx *ctx, float *x, const float *bp, const float *sens, const float *F,
                   float beta, int prior_mode, float sigma2);

/* K1-K6 (BJ configs[0](1)-(3)): frame-integrated model curve F[T][nz][ny][nx] and, if J != NULL,
 * its analytic Jacobian J[4][T][nz][ny][nx] from theta[4][nz][ny][nx].  Evaluated for every voxel (no mask).
 * Rate-dependent scalars are computed in fp64 on the device (fp32 cancels catastrophically).
 * theta outside the box of Q16 is evaluated as given; for k2 + k3 = 0 (below the box: k2 >= 1e-4) F is the limit
 * K1 (1 conv Cp) and dF/dk2, dF/dk3 are returned as 0. */
int kcs_kinetic_eval(kcs_ctx *ctx, const float *theta, float *F, float *J);

/* eq. 4-7 with readings L1-L3, Q12-Q16: n_steps synchronised (Jacobi) Levenberg-Marquardt
 * steps for every in-mask voxel; the Huber gradient uses the previous iterate's 6-neighbourhood.
 * x [T][nz][ny][nx]; theta in/out; lambda in/out (<= 0 -> initialised to 1e-3 max diag J^T J); cost (may be NULL)
 * receives Phi_v after the last step.  Out-of-mask voxels are left untouched (cost 0). */
int kcs_map_lm(kcs_ctx *ctx, const float *x, float *theta, float *lambda, float gamma, float delta,
               int n_steps, float *cost);

/* Options of the fit beyond the hot path, for the kcs_map_lm / kcs_icm_* calls that follow; all
 * pointers [host]; SYNCHRONISES the stream.  opt == NULL restores the defaults (NULL, 6, NULL, 0, NULL, NULL). */
typedef struct {
    const double *frame_weights; /* [T] >= 0: weighted least squares, data term 1/2 sum_m w_m (x_m - F_m)^2 (e.g. frame-duration
                                  * or inverse-variance weights); w_m = 0 drops frame m from the fit */
    int neighbourhood;           /* 6: +-x, +-y, +-z (Q13).  10: the 8 in-plane neighbours of the paper's 3x3 clique (P:114,
                                  * Fig. 1 caption P:47) plus +-z; unit weights, in-volume and in-mask neighbours only */
    const double *delta4;        /* [4] one Huber threshold per parameter map (K1, k2, k3, vB); the scalar delta argument of
                                  * the calls is then ignored */
    int prior_curvature;         /* != 0: the Gauss-Newton curvature of the Huber sum, gamma sum_k H''(xi_p - xi_k,p), joins
                                  * lambda on the diagonal of the LM matrix (eq. 4 as printed has lambda I only) */
    const double *box_lo;        /* [4], [4]: another parameter box than Q16's (both or neither).  lo_p == hi_p FIXES parameter */
    const double *box_hi;        /* p: it sits at lo_p and is not fitted -- k3 in [0, 0] is the one-tissue compartment model */
} kcs_fit_options;
int kcs_set_fit_options(kcs_ctx *ctx, const kcs_fit_options *opt);

/* the macro-parameter map K_i = K1 k3 / (k2 + k3) (net influx rate; 0 where k2 + k3 = 0) from
 * theta[4][nz][ny][nx]; ki[nz][ny][nx] (device).  Evaluated for every voxel. */
int kcs_ki_map(kcs_ctx *ctx, const float *theta, float *ki);

/* P:49 "all effects of attenuation, scatter and randoms".  A frame-independent multiplicative sinogram
 * mult[nz][A][B] (device; attenuation x normalisation factors of every line of response) for the kcs_icm_* calls that
 * follow:   yhat = scale mult (A_s x) + r,   b = scale A_s^T (mult q),   S_s = scale A_s^T mult  (per slice).
 * The library keeps its own copy and builds the S per-slice sensitivity volumes (n_subsets * nz*ny*nx floats of
 * workspace).  NULL restores unit factors.  Scatter is additive: pass randoms + scatter as r with KCS_R_FULL.
 * kcs_forward_project / kcs_back_project / kcs_sensitivity stay the bare operators A, A^T. */
int kcs_set_multiplicative(kcs_ctx *ctx, const float *mult);

/* I: one ICM iteration,
 *   F <- K(theta);  for s = 0..S-1: yhat = scale A_s x + r, q = y/yhat (0 where yhat <= 1e-12),
 *   x <- OSL(x, scale A_s^T q, scale A_s^T 1, F, beta);  theta <- n_lm MAP-LM steps on the new x.
 * y [T][nz][A][B]; r per r_mode (device pointer: r[T] or r[T][nz][A][B]); x, theta, lambda in/out. */
int kcs_icm_iteration(kcs_ctx *ctx, const float *y, const float *r, int r_mode, float scale,
                      float *x, float *theta, float *lambda,
                      float beta, float gamma, float delta, int n_lm);

/* Same iteration, but `n_iter` of them back to back with y packed once (the ICM loop of P:118-125);
 * beta_first is used in the first of them (Q17: 0 when starting from the uniform image). */
int kcs_icm_run(kcs_ctx *ctx, const float *y, const float *r, int r_mode, float scale,
                float *x, float *theta, float *lambda,
                float beta_first, float beta, float gamma, float delta, int n_lm, int n_iter);

/* Host-buffer convenience for end-to-end timing: all data pointers [host] (pinned or pageable); copies
 * y, r, x, theta, lambda to the device, runs kcs_icm_run, copies x, theta, lambda back and synchronises.  x, y and theta
 * move in z chunks on library-owned copy streams beside the OS pass of earlier chunks (alternate chunks on the context's
 * stream and a second library-owned one), theta and lambda return beside the last MAP-LM step; same result as
 * kcs_icm_run, bit for bit. */
int kcs_icm_run_host(kcs_ctx *ctx, const float *y, const float *r, int r_mode, float scale,
                     float *x, float *theta, float *lambda,
                     float beta_first, float beta, float gamma, float delta, int n_lm, int n_iter);

/* ---- the one entry point that allocates nothing ------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): kcs_forward_project (P1-P3, the projection sum of eq. 2's denominator) WITHOUT a kcs_ctx.  It calls no
 * cudaMalloc, cudaFree or allocating library routine: the packed volume, the packed sinogram and the angle table --
 * the workspace kcs_create would allocate -- sit in one static __device__ array of KCS_STATIC_SCRATCH_BYTES inside the
 * library (every GPU this entry point has run on holds that much until the process exits).  The kernels and the
 * arithmetic are those of kcs_forward_project: same result for the same cfg geometry.
 *   cfg     [host] only the geometry is read: nx, ny, nz, vx, vy, n_angles, n_bins, bin_mm, n_steps, step_mm,
 *           n_subsets (frame tables, input function, mask and n_replicas are ignored)
 *   x       [device] nf frames [nf][nz][ny][nx];   y_s [device] out, [nf][nz][As][B], As = A (subset = -1) or A/S
 *   nf      1..KCS_MAX_FRAMES;   stream = the CUDA stream (of the CURRENT device) the work is enqueued on, no sync
 * LIMIT: 256-rounded bytes of  16*2 A  +  4 Tp nz (ny+4)(nx+4)  +  4 Tp nz As B  <= KCS_STATIC_SCRATCH_BYTES
 * (Tp = power of two >= nf, 4..32; BJ configs[0] and [1] fit, configs[2] and [3] do not): a larger problem is rejected
 * with KCS_ERR_SHAPE before any CUDA call, and kcs_static_last_error() says how many bytes it needed.
 * SHARING: every call on a device uses the same array, which keeps the last call's contents (the part that must start
 * at zero is cleared by every call); two calls that overlap on the GPU (different streams, or graphs replayed
 * concurrently) RACE -- order them on one stream or with events.  The first call on a device takes the array's address
 * (cudaGetSymbolAddress, which may load the module): make it outside stream capture.
 * Errors: KCS_ERR_NULL / _SHAPE / _SUBSET / _FRAMES / _CUDA as above; message (per host thread) from
 * kcs_static_last_error(). */
#define KCS_STATIC_SCRATCH_BYTES (40u << 20) /* 40 MiB */
int kcs_forward_project_static(const kcs_config *cfg, const float *x, float *y_s, int subset, int nf, void *stream);
const char *kcs_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
