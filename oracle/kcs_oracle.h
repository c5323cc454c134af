/*
 * kcs_oracle.h -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, fp64 CPU statement of one ICM iteration of Kinetic Compressive
 * Sensing (arXiv 1803.10045, /root/reference/PAPER.md, cited below as P:<line>)
 * with every free choice frozen as in SURVEY.md section 8(c) (readings P1-P5,
 * O1-O2, K1-K6, L1-L3, I, Q1-Q22; also listed in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code with the CUDA
 * path under paper_1803_10045_b200/ and neither includes the other.
 *
 * Parity pins (tests/test_oracle_*.py): projector adjointness and 0/90 degree
 * closed forms; input-function and TAC values at 40 digits; fine-grid and
 * mpmath quadrature of the defining convolution; Jacobian vs central
 * differences; LM noiseless fixed point and brute-force optimum; EM
 * monotonicity; OSEM special cases.  "parity unpinned": the full ICM iterate
 * itself (the paper prints no iterate) beyond those special cases.
 *
 * Layouts (all host pointers, C order, x fastest, double):
 *   activity  x[nf][nz][ny][nx]        sinogram y[nf][nz][A_s][B]
 *   maps  theta[4][nz][ny][nx] in the order (K1, k2, k3, vB)
 */
#ifndef KCS_ORACLE_H
#define KCS_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int nx, ny, nz;
    double vx, vy, vz;          /* voxel size, mm */
    int n_angles, n_bins;       /* theta_a = pi*a/n_angles (Q1) */
    double bin_mm;
    int n_steps;                /* samples per ray (Q3) */
    double step_mm;
    int n_subsets;              /* must divide n_angles; subset s = {a : a mod S == s} (P5) */
    int n_frames;
    const double *t_start_min;  /* [n_frames], minutes */
    const double *t_end_min;
    double feng_A[3];
    double feng_lambda[3];
    const unsigned char *mask;  /* [ny][nx], NULL = Q2 default */
} kcso_config;

#define KCSO_PRIOR_POISSON_MATCHED 0
#define KCSO_PRIOR_ABSOLUTE 1

int kcso_num_threads(void);

/* Q2 default field-of-view mask. */
void kcso_default_mask(const kcso_config *c, unsigned char *mask_out);

/* P1-P3, P5: y = A_s x  (subset < 0: all angles). No scale, no randoms. */
void kcso_forward_project(const kcso_config *c, const double *x, double *y, int subset, int nf);
/* P4: b = A_s^T q, the exact transpose, by scatter. Overwrites b. */
void kcso_back_project(const kcso_config *c, const double *q, double *b, int subset, int nf);
/* A_s^T 1 for one slice, [ny][nx]; (no scale). */
void kcso_sensitivity(const kcso_config *c, int subset, double *sens);

/* O2: x <- M x bp / D for one subset; bp = scale A_s^T q, sens = scale A_s^T 1 ([ny][nx]). */
void kcso_osl_update(const kcso_config *c, double *x, const double *bp, const double *sens,
                     const double *F, double beta, int prior_mode, double sigma2, int nf);

/* K1: Feng input function Cp(t), t in minutes. */
void kcso_input_function(const kcso_config *c, const double *t, int n, double *cp);
/* K2-K6: frame-integrated model curve F[T][V] and Jacobian J[4][T][V] (NULL to skip) for V voxels.
 * theta[4][V].  No mask is applied here. */
void kcso_kinetic_eval(const kcso_config *c, const double *theta, double *F, double *J, long V);
/* pieces exposed for the pins */
double kcso_ICp(const kcso_config *c, double t);                    /* int_0^t Cp */
double kcso_R(const kcso_config *c, double a, double t);             /* (e^{-a.} conv Cp)(t) */
double kcso_G(const kcso_config *c, double a, double t);             /* int_0^t R_a */
double kcso_dGda(const kcso_config *c, double a, double t);
double kcso_Ct(const kcso_config *c, const double xi[4], double t);  /* instantaneous tissue curve */

/* L1: Phi_v(xi) with frozen neighbours nbr[n_nbr][4]. */
double kcso_lm_objective(const kcso_config *c, const double *xv, const double xi[4],
                         const double *nbr, int n_nbr, double gamma, double delta);
/* L2-L3: n_steps synchronised (Jacobi) LM steps on the whole volume. theta, lambda in/out; cost out (may be NULL). */
void kcso_map_lm(const kcso_config *c, const double *x, double *theta, double *lambda,
                 double gamma, double delta, int n_steps, double *cost);

/* S8(f)2 / S8(f)4 options of the fit, oracle-wide (NULL / 6 / NULL restore the hot path of S8(a)):
 * frame_w[n_frames] weights of the data term (weighted least squares); neighbourhood 6 (Q13) or 10 (3x3 in-plane clique
 * of P:114 plus +-z); delta4[4] one Huber threshold per parameter map (the scalar delta argument is then ignored). */
void kcso_set_lm_options(const double *frame_w, int n_frames, int neighbourhood, const double *delta4);

/* second part: prior_curvature != 0 adds gamma sum_k H''(xi_p - xi_k,p) to the diagonal of the LM matrix; box_lo / box_hi
 * (NULL = Q16) replace the parameter box, lo_p == hi_p fixes parameter p (one-tissue model: k3 in [0, 0]). */
void kcso_set_lm_options2(int prior_curvature, const double *box_lo, const double *box_hi);

/* Q15a knob (oracle only): relative slack of the LM acceptance test, default 1e-6. */
void kcso_set_lm_accept_slack(double s);
double kcso_get_lm_accept_slack(void);

/* O1-O2 for all subsets in order 0..S-1 with F held fixed ("one OS-MAP-OSL pass"). r_mode 0: r[T] per-frame
 * constant, 1: r[T][nz][A][B] full sinogram. */
void kcso_os_pass(const kcso_config *c, const double *y, const double *r, int r_mode, double scale,
                  double *x, const double *F, double beta);
/* I: F <- K(theta); OS pass; theta <- L(x, theta, lambda). */
void kcso_icm_iteration(const kcso_config *c, const double *y, const double *r, int r_mode, double scale,
                        double *x, double *theta, double *lambda,
                        double beta, double gamma, double delta, int n_lm);
/* S8(f)3: the same with a multiplicative sinogram mult[nz][A][B] (attenuation x normalisation; NULL = unity):
 * yhat = scale mult (A_s x) + r, b = scale A_s^T (mult q), S_s = scale A_s^T mult (per slice). */
void kcso_os_pass_mult(const kcso_config *c, const double *y, const double *r, int r_mode, double scale, const double *mult,
                       double *x, const double *F, double beta);
void kcso_icm_iteration_mult(const kcso_config *c, const double *y, const double *r, int r_mode, double scale,
                             const double *mult, double *x, double *theta, double *lambda,
                             double beta, double gamma, double delta, int n_lm);

/* K_i = K1 k3 / (k2 + k3) for V voxels, theta[4][V]; 0 where k2 + k3 = 0. */
void kcso_ki_map(const double *theta, double *ki, long V);

/* Poisson log-likelihood sum(y log yhat - yhat), yhat = scale A x + r, all angles (eq. 1 without the prior). */
double kcso_poisson_loglik(const kcso_config *c, const double *y, const double *r, int r_mode,
                           double scale, const double *x);

#ifdef __cplusplus
}
#endif
#endif
