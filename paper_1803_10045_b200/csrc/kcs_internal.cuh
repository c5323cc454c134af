// kcs_internal.cuh -- shared declarations of the CUDA path (not part of the C ABI; see include/kcs.h).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/kcs.h"

// ---------------------------------------------------------------------------------------------
// Geometry handed to kernels by value.
//   padded image layout ("inner"):  xi[z][j+PAD][i+PAD][Tp]  on a (ny+2 PAD) x (nx+2 PAD) grid whose border is 0,
//   so every bilinear tap of a sample with i0 in [-2, nx] is a plain load (P2: outside pixels are 0); the second
//   border pixel lets the forward projector clip rays with a half-pixel margin instead of testing every sample.
//   sinogram layout ("inner"):      qi[z][la][b][Tp]
// ---------------------------------------------------------------------------------------------
#define KCS_PAD 2  // zero pixels around every slice of the padded layout

struct KGeom {
    int nx, ny, nz;    // nz = ALL slices (replicas x slices per replica)
    int nzr;           // slices per replica: z-neighbours exist only inside [k nzr, (k+1) nzr)
    int nxp, nyp;      // nx + 2 KCS_PAD, ny + 2 KCS_PAD
    int A, B, K, S;
    float step_mm, bin_mm;
    double cx, cy, cb, ck;  // (nx-1)/2, (ny-1)/2, (B-1)/2, (K-1)/2
    // per-angle tables (device, double4 each):
    //   fwd[a] = (bin cos/vx, -step sin/vx, bin sin/vy, step cos/vy):  fx = (b-cb) f.x + (k-ck) f.y + cx ; fy = (b-cb) f.z + (k-ck) f.w + cy
    //   bwd[a] = (vx cos/bin, vy sin/bin, -vx sin/step, vy cos/step):  fb = (i-cx) g.x + (j-cy) g.y + cb ; fk = (i-cx) g.z + (j-cy) g.w + ck
    const double4 *fwd;
    const double4 *bwd;
};

// Per-frame kinetic tables (fp64, device).  "b" = value at a frame boundary t (index 0: t_start, 1: t_end).
//   P0[i] = int_0^t e^{-l_i u} du (i = 0..2);  P1_0 = int_0^t u e^{-l_0 u} du;
//   Pn[i-1][n-1] = int_0^t u^n e^{-l_i u} du for i = 1,2 and n = 1..4 (Taylor branch when a ~ l_i).
struct KBoundary {
    double t;
    double P0[3];
    double P1_0;
    double Pn[2][4];
};
struct KFrame {
    KBoundary b[2];
    double dICp;  // int_frame Cp
    double W0;    // int_frame int_0^t Cp  (the a = 0 member of the W family, K3)
    double dt;    // t_end - t_start
    int contiguous;  // t_start == previous frame's t_end (state carried over)
    int new_dt;      // dt differs from the previous frame's (per-duration scalars must be recomputed)
    double w;        // weight of this frame in the least-squares data term (S8(f)4; 1 by default)
};
struct KKin {
    int T;
    double alpha[3];  // K1: Cp(t) = sum (alpha_i + beta_i t) e^{-l_i t}; (alpha, beta) = (-A2-A3, A1), (A2, 0), (A3, 0)
    double beta0;
    double lam[3];
    const KFrame *frames;  // device [T]
};

// Kernel classes for the optional per-kernel timing (kcs_profile_*; bench.py's roofline object).
enum { KCS_K_PACK = 0, KCS_K_UNPACK, KCS_K_KINETIC, KCS_K_FORWARD, KCS_K_BACK, KCS_K_LM, KCS_K_OTHER, KCS_K_NCLASS };
struct KProfRec {
    cudaEvent_t a, b;
    int cls;
};

// A captured kcs_icm_run call (S:7-H6: small problems are launch-bound; a replay is one cudaGraphLaunch).
struct KGraphEntry {
    const void *y, *r, *x, *theta, *lambda;
    int r_mode, n_lm, n_iter;
    float scale, beta_first, beta, gamma, delta;
    cudaStream_t stream;
    long long gen;          // option generation of the context when it was captured
    long long launches;     // kernels inside
    cudaGraphExec_t exec;
};

struct kcs_ctx {
    kcs_config cfg;
    bool prof_on;
    std::vector<KProfRec> prof_recs;     // recorded, not yet read
    std::vector<cudaEvent_t> prof_pool;  // events free for reuse
    std::vector<double> ts, te;
    cudaStream_t stream;
    std::string err;
    long long launches;
    long long ws_bytes;
    bool use_graphs;                    // kcs_use_graphs (default on)
    long long opt_gen, graph_replays;   // bumped by every call that changes what a captured graph bakes in
    std::vector<KGraphEntry> graphs;

    KGeom g;
    KKin kin;
    double4 *d_fwd, *d_bwd;
    KFrame *d_frames;
    std::vector<KFrame> h_frames;     // host copy (kcs_set_fit_options rewrites the frame weights)
    int nbr_mode;                     // 6 (Q13) or 10 (3x3 in-plane clique + the two axial neighbours, S8(f)2)
    bool weighted;                    // some frame weight differs from 1 (S8(f)4)
    bool has_delta4;                  // one Huber threshold per parameter map instead of the scalar argument
    double delta4[4];
    bool prior_curv, custom_box;      // Huber curvature in the LM matrix; a parameter box other than Q16's
    double box_lo[4], box_hi[4];
    unsigned char *d_mask;            // [ny][nx]
    int *d_vlist;                     // in-mask pixel indices j*nx+i of one slice, ascending
    int n_inmask2;                    // their count
    std::vector<unsigned char> h_mask;
    float *d_sens;                    // [S+1][ny][nx], unscaled A_s^T 1; entry S = all angles
    float *d_smax;                    // [S+1] max over the image of d_sens[s]
    float *d_tmp_smax;                // [1] scratch for kcs_osl_update
    // S8(f)3 (kcs_set_multiplicative): n[nz][A][B], unscaled A_s^T n per subset and slice [S][nz][ny][nx], their maxima [S]
    float *d_mult, *d_sens_z, *d_smax_z;
    float4 *d_wtab;                   // back-projector weight table [A][nbj][nbi4][6][4] (k_build_wtab)
    int nbi, nbj, nbi4;               // 2x2 voxel blocks in x, y; groups of 4 blocks in x

    // workspace (inner layouts), sized for Tp = 32
    size_t n_pix_pad;  // nz * nyp * nxp
    size_t n_vox;      // nz * ny * nx
    size_t n_ray_all;  // nz * A * B
    float *xi;   // [n_pix_pad][Tp]
    float *Fi;   // [n_pix_pad][Tp]
    float *qi;   // [n_ray_all][Tp]  (subset or full sinogram being processed)
    float *yi;   // [n_ray_all][Tp]  packed measured data
    float *ri;   // [n_ray_all][Tp]  packed randoms (KCS_R_FULL), allocated lazily
    float *r_pad;  // [32] per-frame randoms padded with 0
    float *theta2;  // [4][n_vox] fp32 scratch for a single Jacobi LM step (the caller's maps cannot be updated in place)
    double *thD[2]; // [4][n_vox] fp64 ping-pong buffers for the steps between the first and the last of a call
    double *lamD;   // [n_vox] lambda in fp64 between those steps
    double *lm_state;  // [15][in-mask voxels] J^T J, J^T r, Phi_data of the current iterate, carried from step to step
    int xi_border_tp;  // Tp for which xi's zero border is valid (0 = unknown)
    float fov_rc2;     // (mask radius + 1.5 voxels)^2, mm^2: rays are clipped to this circle when x is known to be masked

    // device staging buffers of kcs_icm_run_host, allocated lazily
    float *st_y, *st_r, *st_x, *st_theta, *st_lambda;
    size_t st_r_elems;
    cudaStream_t aux_stream;   // kcs_icm_run: the kinetic evaluator runs here beside the first forward projection
    cudaEvent_t ev_fork, ev_join;
    cudaStream_t os_stream;    // second lane of the OS pass (alternate z chunks; kcs_api.cu, icm_run_impl)
    cudaEvent_t ev_os_fork, ev_os_join;
    // kcs_icm_run_host: the volume moves in z chunks; chunk k + 1 is copied in (in_stream) and chunk k - 1 copied out
    // (out_stream) while chunk k goes through its OS pass on the context's stream
    cudaStream_t in_stream, out_stream;
    cudaEvent_t ev_small, ev_lam;          // r / lambda are on the device (theta arrives with the chunks)
    std::vector<cudaEvent_t> ev_in, ev_out;  // per chunk: inputs have arrived / x is final on the device
    std::vector<cudaEvent_t> ev_lm;          // per z piece of the last MAP-LM step: theta, lambda are final on the device
};

#define KCS_CUDA_OK(ctx, call)                                                                  \
    do {                                                                                        \
        cudaError_t e__ = (call);                                                               \
        if (e__ != cudaSuccess) {                                                               \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                   \
            return KCS_ERR_CUDA;                                                                \
        }                                                                                       \
    } while (0)

// Brackets the launches of one kernel class with CUDA events on the context's stream when profiling is on.
struct ProfScope {
    kcs_ctx *c;
    KProfRec r;
    bool live;
    static cudaEvent_t get(kcs_ctx *c) {
        if (!c->prof_pool.empty()) {
            cudaEvent_t e = c->prof_pool.back();
            c->prof_pool.pop_back();
            return e;
        }
        cudaEvent_t e = nullptr;
        cudaEventCreate(&e);
        return e;
    }
    ProfScope(kcs_ctx *ctx, int cls) : c(ctx), live(ctx->prof_on) {
        if (!live) return;
        r.a = get(c); r.b = get(c); r.cls = cls;
        cudaEventRecord(r.a, c->stream);
    }
    ~ProfScope() {
        if (!live) return;
        cudaEventRecord(r.b, c->stream);
        c->prof_recs.push_back(r);
    }
};

// Padded frame count: the power of two >= n (4..32), so that the Tp frames of a pixel (16 Tp / 4 bytes) never
// straddle a 128 B line -- the L1 data pipe charges one wavefront per line touched by a request.
static inline int round_up4(int n) { return n <= 4 ? 4 : n <= 8 ? 8 : n <= 16 ? 16 : 32; }

// ---- launchers (kcs_projector.cu) ----------------------------------------------------------------
// planar [nf][rows][W] (frame stride fs elements)  ->  inner [dst_index(row, col)][Tp]; frames >= nf are written 0.
//   dst_index = (row / rps) * slab + (row % rps) * rstride + off + col
int kcs_launch_pack(kcs_ctx *c, const float *src, size_t fs, int nf, float *dst, int Tp, long long nrows, int W,
                    int rps, long long slab, int rstride, int off);
int kcs_launch_unpack(kcs_ctx *c, const float *src, int Tp, float *dst, size_t fs, int nf, long long nrows, int W,
                      int rps, long long slab, int rstride, int off);
// forward projection of slices [z0, z0 + nzc) of c->xi (Tp frames) for `subset`; out = c->qi.
//   ratio == 0:  qi = step * sum                      (kcs_forward_project)
//   ratio == 1:  qi = y / (scale*step*sum + r), 0 where the denominator <= 1e-12   (O1)
int kcs_launch_forward(kcs_ctx *c, int Tp, int subset, int ratio, float scale, int r_mode, int clip_fov, int z0, int nzc);
// gather back-projection of slices [z0, z0 + nzc) of c->qi for `subset`.
//   osl == 0:  out_inner (padded layout) = step * sum                              (kcs_back_project)
//   osl == 1:  c->xi <- OSL update with bp = scale*step*sum, sens = scale*A_s^T 1, F = c->Fi   (O2)
int kcs_launch_back(kcs_ctx *c, int Tp, int subset, int osl, float *out_inner, float scale, float beta, int z0, int nzc);
int kcs_launch_sens(kcs_ctx *c);  // fills d_sens, d_smax
int kcs_launch_subset_rows(kcs_ctx *c, const float *n, float *out, int s);  // out[z][la][b] = n[z][s + la S][b]
int kcs_launch_max_nonneg(kcs_ctx *c, const float *v, size_t n, float *out);  // *out = max(0, max v)
int kcs_launch_build_wtab(kcs_ctx *c);  // fills d_wtab
int kcs_launch_osl_planar(kcs_ctx *c, float *x, const float *bp, const float *sens, const float *F, float beta,
                          int prior_mode, float sigma2);

// ---- launchers (kcs_kinetic.cu) ------------------------------------------------------------------
// F (and J) from theta.  inner == 0: F planar [T][V], J planar [4][T][V] or NULL;  inner == 1: F = padded inner layout, Tp.
// (z0, nzc): slices [z0, z0 + nzc) only (inner == 1, J == NULL); nzc < 0 = up to the last slice.
int kcs_launch_kinetic(kcs_ctx *c, const float *theta, float *F, float *J, int inner, int Tp, int z0 = 0, int nzc = -1);
int kcs_launch_ki_map(kcs_ctx *c, const float *theta, float *ki);
// one Jacobi LM step: reads theta_in, writes theta_out for the in-mask voxels (masked-out voxels are never touched).
//   x_inner == 0: x planar [T][V];  x_inner == 1: x = c->xi padded inner layout with Tp.
int kcs_launch_lm_step(kcs_ctx *c, const float *x, int x_inner, int Tp, const void *theta_in, int in_f64, void *theta_out,
                       int out_f64, const void *lam_in, void *lam_out, float gamma, float delta, float *cost, int z0 = 0,
                       int nzc = -1);  // slices [z0, z0 + nzc) only (Jacobi: a step reads theta_in, so z ranges are independent)
