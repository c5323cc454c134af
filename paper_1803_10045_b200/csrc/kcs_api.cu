// kcs_api.cu -- the C ABI of include/kcs.h: argument checking, context set-up (geometry and kinetic tables in
// fp64 on the host), and the sequencing of kernels for each entry point.  No compute happens on the host.
#include <climits>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "kcs_internal.cuh"

namespace {

thread_local std::string g_create_err;

int fail(kcs_ctx *c, int code, const std::string &msg) {
    if (c) c->err = msg;
    else g_create_err = msg;
    return code;
}

// ---- host quadrature for the voxel-independent kinetic tables (K3, K4) -------------------------------
// 8-point Gauss-Legendre on `panels` equal panels; every integrand here is entire, so this is exact to rounding.
template <class F>
long double gl8(F f, long double a, long double b, int panels) {
    static const long double xs[4] = {0.1834346424956498049L, 0.5255324099163289858L, 0.7966664774136267396L,
                                      0.9602898564975362317L};
    static const long double ws[4] = {0.3626837833783619830L, 0.3137066458778872873L, 0.2223810344533744706L,
                                      0.1012285362903762591L};
    if (!(b > a)) return 0.0L;
    const long double h = (b - a) / panels;
    long double sum = 0.0L;
    for (int p = 0; p < panels; ++p) {
        const long double mid = a + (p + 0.5L) * h, half = 0.5L * h;
        long double s = 0.0L;
        for (int q = 0; q < 4; ++q) s += ws[q] * (f(mid - half * xs[q]) + f(mid + half * xs[q]));
        sum += s * half;
    }
    return sum;
}

int panels_for(long double len) {
    int p = (int)std::ceil((double)len * 16.0);
    return p < 64 ? 64 : p;
}

struct Feng {
    long double al[3], be[3], lam[3];
    long double Cp(long double t) const {
        long double s = 0.0L;
        for (int i = 0; i < 3; ++i) s += (al[i] + be[i] * t) * expl(-lam[i] * t);
        return s;
    }
};

void fill_boundary(const Feng &fe, double t, KBoundary &b) {
    b.t = t;
    const int np = panels_for(t);
    for (int i = 0; i < 3; ++i) {
        const long double l = fe.lam[i];
        b.P0[i] = (double)gl8([&](long double u) { return expl(-l * u); }, 0.0L, t, np);
    }
    {
        const long double l = fe.lam[0];
        b.P1_0 = (double)gl8([&](long double u) { return u * expl(-l * u); }, 0.0L, t, np);
    }
    for (int i = 1; i < 3; ++i) {
        const long double l = fe.lam[i];
        for (int n = 1; n <= 4; ++n)
            b.Pn[i - 1][n - 1] = (double)gl8([&](long double u) { return powl(u, n) * expl(-l * u); }, 0.0L, t, np);
    }
}

int check_cfg(const kcs_config *c, std::string &why) {
    if (c->nx <= 0 || c->ny <= 0 || c->nz <= 0 || c->n_angles <= 0 || c->n_bins < 5 || c->n_steps <= 0 ||
        c->n_subsets <= 0 || c->n_replicas < 0 || !(c->vx > 0) || !(c->vy > 0) || !(c->bin_mm > 0) || !(c->step_mm > 0)) {
        why = "non-positive size (n_bins must be >= 5: the back-projector reads 5-bin windows)";
        return KCS_ERR_SHAPE;
    }
    if (c->n_angles % c->n_subsets != 0) {
        why = "n_subsets does not divide n_angles";
        return KCS_ERR_SUBSET;
    }
    if (c->n_frames <= 0 || c->n_frames > KCS_MAX_FRAMES) {
        why = "n_frames must be in [1, KCS_MAX_FRAMES]";
        return KCS_ERR_FRAMES;
    }
    if (!c->t_start_min || !c->t_end_min) {
        why = "frame tables are NULL";
        return KCS_ERR_NULL;
    }
    for (int m = 0; m < c->n_frames; ++m)
        if (!(c->t_end_min[m] > c->t_start_min[m]) || c->t_start_min[m] < 0.0) {
            why = "frame with t_end <= t_start or negative start";
            return KCS_ERR_FRAMES;
        }
    for (int i = 0; i < 3; ++i)
        if (!(c->feng_lambda[i] > 0.f)) {
            why = "feng_lambda must be positive";
            return KCS_ERR_SHAPE;
        }
    // the evaluator divides by a - lambda_1 without a series branch: lambda_1 must lie outside the rate box a = k2 + k3 <= 3 (Q16)
    if (!(c->feng_lambda[0] > 3.05f)) {
        why = "feng_lambda[0] must exceed 3.05 (it may not fall inside the rate box k2 + k3 <= 3)";
        return KCS_ERR_SHAPE;
    }
    for (int a = 0; a < c->n_angles; ++a) {
        const double th = M_PI * a / c->n_angles, cs = std::fabs(std::cos(th)), sn = std::fabs(std::sin(th));
        if ((cs * c->vx + sn * c->vy) / c->bin_mm > 1.5 || (sn * c->vx + cs * c->vy) / c->step_mm > 1.5) {
            why = "voxel too large for the bin/step size: a voxel would see more than 3x3 ray samples per angle";
            return KCS_ERR_SHAPE;
        }
    }
    return KCS_OK;
}

template <class T>
cudaError_t dalloc(kcs_ctx *c, T **p, size_t n) {
    cudaError_t e = cudaMalloc((void **)p, n * sizeof(T));
    if (e == cudaSuccess) c->ws_bytes += (long long)(n * sizeof(T));
    return e;
}

int ensure_border(kcs_ctx *c, int Tp) {
    if (c->xi_border_tp != Tp) {
        KCS_CUDA_OK(c, cudaMemsetAsync(c->xi, 0, c->n_pix_pad * (size_t)Tp * sizeof(float), c->stream));
        c->xi_border_tp = Tp;
    }
    return KCS_OK;
}

// slices [z0, z0 + nzc) of a planar image [nf][nz][ny][nx]  <->  the padded frame-innermost layout
int pack_image(kcs_ctx *c, const float *planar, int nf, float *inner, int Tp, int z0 = 0, int nzc = -1) {
    const KGeom &g = c->g;
    if (nzc < 0) nzc = g.nz;
    return kcs_launch_pack(c, planar + (size_t)z0 * g.ny * g.nx, c->n_vox, nf, inner + (size_t)z0 * g.nyp * g.nxp * Tp, Tp,
                           (long long)nzc * g.ny, g.nx, g.ny, (long long)g.nyp * g.nxp, g.nxp, KCS_PAD * (g.nxp + 1));
}
int unpack_image(kcs_ctx *c, const float *inner, int Tp, float *planar, int nf, int z0 = 0, int nzc = -1) {
    const KGeom &g = c->g;
    if (nzc < 0) nzc = g.nz;
    return kcs_launch_unpack(c, inner + (size_t)z0 * g.nyp * g.nxp * Tp, Tp, planar + (size_t)z0 * g.ny * g.nx, c->n_vox, nf,
                             (long long)nzc * g.ny, g.nx, g.ny, (long long)g.nyp * g.nxp, g.nxp, KCS_PAD * (g.nxp + 1));
}
int pack_sino(kcs_ctx *c, const float *planar, int nf, float *inner, int Tp, int As, int z0 = 0, int nzc = -1) {
    const KGeom &g = c->g;
    if (nzc < 0) nzc = g.nz;
    return kcs_launch_pack(c, planar + (size_t)z0 * As * g.B, (size_t)g.nz * As * g.B, nf, inner + (size_t)z0 * As * g.B * Tp, Tp,
                           (long long)nzc * As, g.B, INT_MAX, 0, g.B, 0);
}
int unpack_sino(kcs_ctx *c, const float *inner, int Tp, float *planar, int nf, int As) {
    const KGeom &g = c->g;
    return kcs_launch_unpack(c, inner, Tp, planar, (size_t)g.nz * As * g.B, nf, (long long)g.nz * As, g.B, INT_MAX, 0, g.B,
                             0);
}

int check_subset_frames(kcs_ctx *c, int subset, int f0, int nf) {
    if (subset < -1 || subset >= c->cfg.n_subsets) return fail(c, KCS_ERR_SHAPE, "subset out of range");
    if (f0 < 0 || nf <= 0 || f0 + nf > c->cfg.n_frames) return fail(c, KCS_ERR_SHAPE, "frame range out of [0, n_frames)");
    return KCS_OK;
}

}  // namespace

extern "C" {

const char *kcs_last_error(const kcs_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

long long kcs_workspace_bytes(const kcs_ctx *ctx) { return ctx ? ctx->ws_bytes : 0; }
long long kcs_launch_count(const kcs_ctx *ctx) { return ctx ? ctx->launches : 0; }

int kcs_set_stream(kcs_ctx *ctx, void *stream) {
    if (!ctx) return KCS_ERR_NULL;
    ctx->stream = (cudaStream_t)stream;
    return KCS_OK;
}

int kcs_use_graphs(kcs_ctx *c, int on) {
    if (!c) return KCS_ERR_NULL;
    c->use_graphs = on != 0;
    return KCS_OK;
}
long long kcs_graph_replays(const kcs_ctx *ctx) { return ctx ? ctx->graph_replays : 0; }

int kcs_profile_enable(kcs_ctx *c, int on) {
    if (!c) return KCS_ERR_NULL;
    c->prof_on = on != 0;
    return KCS_OK;
}

int kcs_profile_read(kcs_ctx *c, double *ms, long long *count, int n_classes) {
    if (!c) return KCS_ERR_NULL;
    if (!ms || !count) return fail(c, KCS_ERR_NULL, "kcs_profile_read: NULL buffer");
    if (n_classes < KCS_PROFILE_NCLASS) return fail(c, KCS_ERR_SHAPE, "kcs_profile_read: n_classes < KCS_PROFILE_NCLASS");
    for (int q = 0; q < n_classes; ++q) { ms[q] = 0.0; count[q] = 0; }
    KCS_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    for (const KProfRec &r : c->prof_recs) {
        float t = 0.f;
        KCS_CUDA_OK(c, cudaEventElapsedTime(&t, r.a, r.b));
        ms[r.cls] += (double)t;
        count[r.cls] += 1;
        c->prof_pool.push_back(r.a);
        c->prof_pool.push_back(r.b);
    }
    c->prof_recs.clear();
    return KCS_OK;
}

int kcs_get_mask(const kcs_ctx *ctx, unsigned char *out) {
    if (!ctx || !out) return KCS_ERR_NULL;
    std::memcpy(out, ctx->h_mask.data(), ctx->h_mask.size());
    return KCS_OK;
}

int kcs_destroy(kcs_ctx *c) {
    if (!c) return KCS_ERR_NULL;
    cudaStreamSynchronize(c->stream);
    void *ptrs[] = {c->d_mult, c->d_sens_z, c->d_smax_z, c->d_fwd, c->d_bwd, c->d_frames, c->d_mask, c->d_sens, c->d_smax, c->d_tmp_smax, c->d_wtab, c->d_vlist, c->xi, c->Fi,
                    c->qi, c->yi, c->ri, c->r_pad, c->theta2, c->thD[0], c->thD[1], c->lamD, c->lm_state, c->st_y, c->st_r, c->st_x, c->st_theta, c->st_lambda};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    for (KGraphEntry &ge : c->graphs) cudaGraphExecDestroy(ge.exec);
    for (const KProfRec &r : c->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (cudaEvent_t e : c->prof_pool) cudaEventDestroy(e);
    if (c->in_stream) { cudaStreamDestroy(c->in_stream); cudaStreamDestroy(c->out_stream); cudaEventDestroy(c->ev_small); cudaEventDestroy(c->ev_lam); }
    for (cudaEvent_t e : c->ev_in) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_out) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_lm) cudaEventDestroy(e);
    if (c->aux_stream) { cudaStreamDestroy(c->aux_stream); cudaEventDestroy(c->ev_fork); cudaEventDestroy(c->ev_join); }
    if (c->os_stream) { cudaStreamDestroy(c->os_stream); cudaEventDestroy(c->ev_os_fork); cudaEventDestroy(c->ev_os_join); }
    delete c;
    return KCS_OK;
}

int kcs_create(kcs_ctx **out, const kcs_config *cfg, void *stream) {
    if (!out || !cfg) return fail(nullptr, KCS_ERR_NULL, "kcs_create: NULL argument");
    *out = nullptr;
    std::string why;
    int rc = check_cfg(cfg, why);
    if (rc != KCS_OK) return fail(nullptr, rc, "kcs_create: " + why);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, KCS_ERR_CUDA, "kcs_create: no CUDA device (this library has no CPU fallback)");
    }
    kcs_ctx *c = new (std::nothrow) kcs_ctx();
    if (!c) return fail(nullptr, KCS_ERR_ALLOC, "kcs_create: host allocation failed");
    c->cfg = *cfg;
    c->ts.assign(cfg->t_start_min, cfg->t_start_min + cfg->n_frames);
    c->te.assign(cfg->t_end_min, cfg->t_end_min + cfg->n_frames);
    c->cfg.t_start_min = c->ts.data();
    c->cfg.t_end_min = c->te.data();
    c->cfg.mask_host = nullptr;
    c->stream = (cudaStream_t)stream;
    c->launches = 0;
    c->ws_bytes = 0;
    c->use_graphs = true;
    c->opt_gen = 0;
    c->graph_replays = 0;
    c->prof_on = false;
    c->xi_border_tp = 0;
    c->d_fwd = c->d_bwd = nullptr; c->d_frames = nullptr; c->d_mask = nullptr;
    c->d_sens = c->d_smax = c->d_tmp_smax = nullptr;
    c->d_mult = c->d_sens_z = c->d_smax_z = nullptr;
    c->d_wtab = nullptr;
    c->d_vlist = nullptr; c->n_inmask2 = 0;
    c->xi = c->Fi = c->qi = c->yi = c->ri = c->r_pad = c->theta2 = nullptr;
    c->thD[0] = c->thD[1] = c->lamD = nullptr;
    c->lm_state = nullptr;
    c->in_stream = c->out_stream = nullptr; c->ev_small = c->ev_lam = nullptr;
    c->aux_stream = nullptr; c->ev_fork = c->ev_join = nullptr;
    c->os_stream = nullptr; c->ev_os_fork = c->ev_os_join = nullptr;
    c->st_y = c->st_r = c->st_x = c->st_theta = c->st_lambda = nullptr;
    c->st_r_elems = 0;

    const int nrep = cfg->n_replicas > 0 ? cfg->n_replicas : 1;
    const int nx = cfg->nx, ny = cfg->ny, nz = cfg->nz * nrep, A = cfg->n_angles, B = cfg->n_bins, K = cfg->n_steps, T = cfg->n_frames;
    KGeom &g = c->g;
    g.nx = nx; g.ny = ny; g.nz = nz; g.nzr = cfg->nz; g.nxp = nx + 2 * KCS_PAD; g.nyp = ny + 2 * KCS_PAD;
    g.A = A; g.B = B; g.K = K; g.S = cfg->n_subsets;
    g.step_mm = cfg->step_mm; g.bin_mm = cfg->bin_mm;
    g.cx = 0.5 * (nx - 1); g.cy = 0.5 * (ny - 1); g.cb = 0.5 * (B - 1); g.ck = 0.5 * (K - 1);
    c->n_vox = (size_t)nz * ny * nx;
    c->n_pix_pad = (size_t)nz * g.nyp * g.nxp;
    c->n_ray_all = (size_t)nz * A * B;

    // P1: angle tables (fp64)
    std::vector<double4> fw(A), bw(A);
    for (int a = 0; a < A; ++a) {
        const double th = M_PI * (double)a / (double)A, cs = std::cos(th), sn = std::sin(th);
        const double vx = cfg->vx, vy = cfg->vy, bin = cfg->bin_mm, st = cfg->step_mm;
        fw[a] = make_double4(bin * cs / vx, -st * sn / vx, bin * sn / vy, st * cs / vy);
        bw[a] = make_double4(vx * cs / bin, vy * sn / bin, -vx * sn / st, vy * cs / st);
    }
    // Q2: field-of-view mask
    c->h_mask.resize((size_t)nx * ny);
    if (cfg->mask_host) {
        for (size_t q = 0; q < c->h_mask.size(); ++q) c->h_mask[q] = cfg->mask_host[q] ? 1 : 0;
    } else {
        int mn = nx < ny ? nx : ny;
        if (B < mn) mn = B;
        if (K < mn) mn = K;
        const double rad = (0.5 * mn - 1.0) * cfg->vx;
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const double X = (i - g.cx) * cfg->vx, Y = (j - g.cy) * cfg->vy;
                c->h_mask[(size_t)j * nx + i] = (X * X + Y * Y <= rad * rad) ? 1 : 0;
            }
    }
    {   // radius of the smallest centred circle that holds every in-mask voxel centre, plus 1.5 voxels for the taps
        double r2 = 0.0;
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                if (c->h_mask[(size_t)j * nx + i]) {
                    const double X = (i - g.cx) * cfg->vx, Y = (j - g.cy) * cfg->vy;
                    if (X * X + Y * Y > r2) r2 = X * X + Y * Y;
                }
        const double rc = std::sqrt(r2) + 1.5 * (cfg->vx > cfg->vy ? cfg->vx : cfg->vy);
        c->fov_rc2 = (float)(rc * rc);
    }
    // K1, K3, K4: kinetic tables (fp64 via long-double quadrature)
    Feng fe;
    fe.al[0] = -(long double)cfg->feng_A[1] - (long double)cfg->feng_A[2];
    fe.be[0] = cfg->feng_A[0];
    fe.al[1] = cfg->feng_A[1]; fe.be[1] = 0.0L;
    fe.al[2] = cfg->feng_A[2]; fe.be[2] = 0.0L;
    for (int i = 0; i < 3; ++i) fe.lam[i] = cfg->feng_lambda[i];
    std::vector<KFrame> frames(T);
    for (int m = 0; m < T; ++m) {
        KFrame &f = frames[m];
        const double ts = c->ts[m], te = c->te[m];
        fill_boundary(fe, ts, f.b[0]);
        fill_boundary(fe, te, f.b[1]);
        f.dt = te - ts;
        const long double ICp_ts = gl8([&](long double u) { return fe.Cp(u); }, 0.0L, ts, panels_for(ts));
        const int np = panels_for(f.dt);
        f.dICp = (double)gl8([&](long double u) { return fe.Cp(u); }, ts, te, np);
        // W0 = int_ts^te ICp(t) dt = dt ICp(ts) + int_ts^te (te - u) Cp(u) du
        f.W0 = (double)((long double)f.dt * ICp_ts +
                        gl8([&](long double u) { return ((long double)te - u) * fe.Cp(u); }, ts, te, np));
        f.contiguous = (m > 0 && c->ts[m] == c->te[m - 1]) ? 1 : 0;
        f.w = 1.0;
        if (m > 0 && std::fabs(f.dt - frames[m - 1].dt) <= 1e-12 * f.dt) {
            f.dt = frames[m - 1].dt;  // same duration class: per-duration scalars are reused (1e-12 relative)
            f.new_dt = 0;
        } else {
            f.new_dt = 1;
        }
    }
    KKin &kin = c->kin;
    kin.T = T;
    for (int i = 0; i < 3; ++i) {
        kin.alpha[i] = (double)fe.al[i];
        kin.lam[i] = (double)fe.lam[i];
    }
    kin.beta0 = (double)fe.be[0];
    c->h_frames = frames;
    c->nbr_mode = 6;
    c->has_delta4 = false;
    c->weighted = false;
    c->prior_curv = c->custom_box = false;
    { const double lo[4] = {0.0, 1e-4, 0.0, 0.0}, hi[4] = {2.0, 2.0, 1.0, 1.0};  // Q16
      for (int p = 0; p < 4; ++p) { c->box_lo[p] = lo[p]; c->box_hi[p] = hi[p]; } }

    std::vector<int> vlist;
    for (int q = 0; q < nx * ny; ++q)
        if (c->h_mask[q]) vlist.push_back(q);
    c->n_inmask2 = (int)vlist.size();
    vlist.resize((size_t)nx * ny, 0);
    const int Tp = round_up4(T);
    c->nbi = (nx + 1) / 2; c->nbj = (ny + 1) / 2; c->nbi4 = (c->nbi + 3) / 4;
    cudaError_t e = cudaSuccess;
#define TRY(x) if (e == cudaSuccess) e = (x)
    TRY(dalloc(c, &c->d_fwd, (size_t)A));
    TRY(dalloc(c, &c->d_bwd, (size_t)A));
    TRY(dalloc(c, &c->d_frames, (size_t)T));
    TRY(dalloc(c, &c->d_mask, (size_t)nx * ny));
    TRY(dalloc(c, &c->d_vlist, (size_t)nx * ny));
    TRY(dalloc(c, &c->d_sens, (size_t)(g.S + 1) * nx * ny));
    TRY(dalloc(c, &c->d_smax, (size_t)g.S + 1));
    TRY(dalloc(c, &c->d_tmp_smax, (size_t)1));
    TRY(dalloc(c, &c->d_wtab, (size_t)A * c->nbj * c->nbi4 * 24));
    TRY(dalloc(c, &c->xi, c->n_pix_pad * Tp));
    TRY(dalloc(c, &c->Fi, c->n_pix_pad * Tp));
    TRY(dalloc(c, &c->qi, c->n_ray_all * Tp));
    TRY(dalloc(c, &c->yi, c->n_ray_all * Tp));
    TRY(dalloc(c, &c->r_pad, (size_t)KCS_MAX_FRAMES));
    TRY(dalloc(c, &c->theta2, 4 * c->n_vox));
    TRY(dalloc(c, &c->thD[0], 4 * c->n_vox));
    TRY(dalloc(c, &c->thD[1], 4 * c->n_vox));
    TRY(dalloc(c, &c->lamD, c->n_vox));
    TRY(dalloc(c, &c->lm_state, (size_t)15 * (size_t)c->n_inmask2 * nz + 1));
    TRY(cudaMemcpyAsync(c->d_fwd, fw.data(), sizeof(double4) * A, cudaMemcpyHostToDevice, c->stream));
    TRY(cudaMemcpyAsync(c->d_bwd, bw.data(), sizeof(double4) * A, cudaMemcpyHostToDevice, c->stream));
    TRY(cudaMemcpyAsync(c->d_frames, frames.data(), sizeof(KFrame) * T, cudaMemcpyHostToDevice, c->stream));
    TRY(cudaMemcpyAsync(c->d_mask, c->h_mask.data(), (size_t)nx * ny, cudaMemcpyHostToDevice, c->stream));
    TRY(cudaMemcpyAsync(c->d_vlist, vlist.data(), sizeof(int) * vlist.size(), cudaMemcpyHostToDevice, c->stream));
    TRY(cudaMemsetAsync(c->Fi, 0, c->n_pix_pad * Tp * sizeof(float), c->stream));
#undef TRY
    if (e != cudaSuccess) {
        const bool oom = (e == cudaErrorMemoryAllocation);
        std::string msg = std::string("kcs_create: ") + cudaGetErrorString(e);
        cudaGetLastError();
        kcs_destroy(c);
        return fail(nullptr, oom ? KCS_ERR_ALLOC : KCS_ERR_CUDA, msg);
    }
    g.fwd = c->d_fwd;
    g.bwd = c->d_bwd;
    kin.frames = c->d_frames;
    rc = kcs_launch_sens(c);
    if (rc == KCS_OK) rc = kcs_launch_build_wtab(c);
    if (rc == KCS_OK && cudaStreamSynchronize(c->stream) != cudaSuccess) rc = KCS_ERR_CUDA;
    if (rc != KCS_OK) {
        std::string msg = "kcs_create: sensitivity kernel failed: " + c->err;
        kcs_destroy(c);
        return fail(nullptr, rc, msg);
    }
    *out = c;
    return KCS_OK;
}

int kcs_forward_project(kcs_ctx *c, const float *x, float *y_s, int subset, int f0, int nf) {
    if (!c) return KCS_ERR_NULL;
    if (!x || !y_s) return fail(c, KCS_ERR_NULL, "kcs_forward_project: NULL buffer");
    int rc = check_subset_frames(c, subset, f0, nf);
    if (rc) return rc;
    const KGeom &g = c->g;
    const int Tp = round_up4(nf), As = subset < 0 ? g.A : g.A / g.S;
    if ((rc = ensure_border(c, Tp))) return rc;
    if ((rc = pack_image(c, x + (size_t)f0 * c->n_vox, nf, c->xi, Tp))) return rc;
    if ((rc = kcs_launch_forward(c, Tp, subset, 0, 1.f, 0, 0, 0, g.nz))) return rc;
    return unpack_sino(c, c->qi, Tp, y_s + (size_t)f0 * g.nz * As * g.B, nf, As);
}

int kcs_back_project(kcs_ctx *c, const float *q_s, float *b, int subset, int f0, int nf) {
    if (!c) return KCS_ERR_NULL;
    if (!q_s || !b) return fail(c, KCS_ERR_NULL, "kcs_back_project: NULL buffer");
    int rc = check_subset_frames(c, subset, f0, nf);
    if (rc) return rc;
    const KGeom &g = c->g;
    const int Tp = round_up4(nf), As = subset < 0 ? g.A : g.A / g.S;
    if ((rc = ensure_border(c, Tp))) return rc;
    if ((rc = pack_sino(c, q_s + (size_t)f0 * g.nz * As * g.B, nf, c->qi, Tp, As))) return rc;
    if ((rc = kcs_launch_back(c, Tp, subset, 0, c->xi, 1.f, 0.f, 0, g.nz))) return rc;
    return unpack_image(c, c->xi, Tp, b + (size_t)f0 * c->n_vox, nf);
}

int kcs_sensitivity(kcs_ctx *c, int subset, float *sens) {
    if (!c) return KCS_ERR_NULL;
    if (!sens) return fail(c, KCS_ERR_NULL, "kcs_sensitivity: NULL buffer");
    if (subset < -1 || subset >= c->g.S) return fail(c, KCS_ERR_SHAPE, "subset out of range");
    const size_t v2 = (size_t)c->g.nx * c->g.ny;
    const int sidx = subset < 0 ? c->g.S : subset;
    KCS_CUDA_OK(c, cudaMemcpyAsync(sens, c->d_sens + sidx * v2, v2 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    return KCS_OK;
}

// S8(f)3: the sensitivity images A_s^T n are one plain back-projection of n (as a one-frame sinogram) per subset.
int kcs_set_multiplicative(kcs_ctx *c, const float *mult) {
    if (!c) return KCS_ERR_NULL;
    c->opt_gen++;
    const KGeom &g = c->g;
    if (!mult) {  // back to unit factors
        if (c->d_mult) { cudaStreamSynchronize(c->stream); cudaFree(c->d_mult); c->d_mult = nullptr; }
        return KCS_OK;
    }
    const size_t nr = c->n_ray_all, nv = c->n_vox;
    cudaError_t e = cudaSuccess;
    if (!c->d_mult) {
        e = dalloc(c, &c->d_mult, nr);
        if (e == cudaSuccess && !c->d_sens_z) e = dalloc(c, &c->d_sens_z, (size_t)g.S * nv);
        if (e == cudaSuccess && !c->d_smax_z) e = dalloc(c, &c->d_smax_z, (size_t)g.S);
        if (e != cudaSuccess) {
            cudaGetLastError();
            if (c->d_mult) { cudaFree(c->d_mult); c->d_mult = nullptr; }
            return fail(c, KCS_ERR_ALLOC, "kcs_set_multiplicative: cannot allocate the per-slice sensitivity images");
        }
    }
    KCS_CUDA_OK(c, cudaMemcpyAsync(c->d_mult, mult, nr * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    const int Tp = 4, As = g.A / g.S;
    int rc;
    if ((rc = ensure_border(c, Tp))) return rc;
    float *rows = c->yi;  // scratch: the packed-data buffer is rewritten by the next kcs_icm_* call anyway
    for (int s = 0; s < g.S; ++s) {
        if ((rc = kcs_launch_subset_rows(c, c->d_mult, rows, s))) return rc;
        if ((rc = pack_sino(c, rows, 1, c->qi, Tp, As))) return rc;
        if ((rc = kcs_launch_back(c, Tp, s, 0, c->xi, 1.f, 0.f, 0, g.nz))) return rc;
        if ((rc = unpack_image(c, c->xi, Tp, c->d_sens_z + (size_t)s * nv, 1))) return rc;
        if ((rc = kcs_launch_max_nonneg(c, c->d_sens_z + (size_t)s * nv, nv, c->d_smax_z + s))) return rc;
    }
    return KCS_OK;
}

int kcs_osl_update(kcs_ctx *c, float *x, const float *bp, const float *sens, const float *F, float beta, int prior_mode,
                   float sigma2) {
    if (!c) return KCS_ERR_NULL;
    if (!x || !bp || !sens || !F) return fail(c, KCS_ERR_NULL, "kcs_osl_update: NULL buffer");
    if (prior_mode != KCS_PRIOR_POISSON_MATCHED && prior_mode != KCS_PRIOR_ABSOLUTE)
        return fail(c, KCS_ERR_SHAPE, "kcs_osl_update: unknown prior_mode");
    if (prior_mode == KCS_PRIOR_ABSOLUTE && !(sigma2 > 0.f)) return fail(c, KCS_ERR_SHAPE, "kcs_osl_update: sigma2 <= 0");
    return kcs_launch_osl_planar(c, x, bp, sens, F, beta, prior_mode, sigma2);
}

int kcs_ki_map(kcs_ctx *c, const float *theta, float *ki) {
    if (!c) return KCS_ERR_NULL;
    if (!theta || !ki) return fail(c, KCS_ERR_NULL, "kcs_ki_map: NULL buffer");
    return kcs_launch_ki_map(c, theta, ki);
}

int kcs_kinetic_eval(kcs_ctx *c, const float *theta, float *F, float *J) {
    if (!c) return KCS_ERR_NULL;
    if (!theta || !F) return fail(c, KCS_ERR_NULL, "kcs_kinetic_eval: NULL buffer");
    return kcs_launch_kinetic(c, theta, F, J, 0, 0);
}

// n_steps Jacobi steps.  The first reads the caller's fp32 maps, the last writes them; in between the iterate lives
// in the context's fp64 ping-pong buffers, so a call rounds theta and lambda to fp32 once, not once per step.
// Host-buffer mode of the ICM loop (kcs_icm_run_host): y, x and theta arrive from / x, theta, lambda return to HOST memory in
// z ranges.
#define KCS_MAX_CHUNKS 9
#define KCS_LM_PIECES 4
struct HostIO {
    const float *hy;   // [host] y[T][nz][A][B]
    float *hx;         // [host] x[T][nz][ny][nx], in and out
    int nchunk;
    int zb[KCS_MAX_CHUNKS + 1];  // chunk k = slices [zb[k], zb[k + 1])
    cudaEvent_t ev_lam;          // lambda (copied in last: only MAP-LM reads it) is on the device
    // the last MAP-LM step of the call runs in z pieces, so that theta and lambda of a piece leave while the next is fitted
    int n_piece;                 // set by lm_steps: 0 = the step was not split
    int pzb[KCS_LM_PIECES + 1];
    cudaEvent_t ev_lm[KCS_LM_PIECES];
};

static int lm_steps(kcs_ctx *c, const float *x, int x_inner, int Tp, float *theta, float *lambda, float gamma, float delta,
                    int n_steps, float *cost, HostIO *io = nullptr) {
    const size_t map_bytes = 4 * c->n_vox * sizeof(float);
    if (cost) KCS_CUDA_OK(c, cudaMemsetAsync(cost, 0, c->n_vox * sizeof(float), c->stream));  // out-of-mask voxels: 0
    if (n_steps == 1) {  // fp32 scratch pre-filled with the caller's maps: the kernel only writes in-mask voxels
        KCS_CUDA_OK(c, cudaMemcpyAsync(c->theta2, theta, map_bytes, cudaMemcpyDeviceToDevice, c->stream));
        int rc = kcs_launch_lm_step(c, x, x_inner, Tp, theta, 0, c->theta2, 0, lambda, lambda, gamma, delta, cost);
        if (rc) return rc;
        KCS_CUDA_OK(c, cudaMemcpyAsync(theta, c->theta2, map_bytes, cudaMemcpyDeviceToDevice, c->stream));
        return KCS_OK;
    }
    for (int s = 0; s < n_steps; ++s) {
        const bool first = s == 0, last = s == n_steps - 1;
        const void *tin = first ? (const void *)theta : (const void *)c->thD[(s + 1) & 1];
        void *tout = last ? (void *)theta : (void *)c->thD[s & 1];
        const void *lin = first ? (const void *)lambda : (const void *)c->lamD;
        void *lout = last ? (void *)lambda : (void *)c->lamD;
        if (last && io && c->g.nz >= KCS_LM_PIECES) {  // Jacobi: the step reads tin only, z pieces are independent launches
            io->n_piece = KCS_LM_PIECES;
            for (int p = 0; p <= KCS_LM_PIECES; ++p) io->pzb[p] = (int)((long long)c->g.nz * p / KCS_LM_PIECES);
            for (int p = 0; p < KCS_LM_PIECES; ++p) {
                int rc = kcs_launch_lm_step(c, x, x_inner, Tp, tin, 1, tout, 0, lin, lout, gamma, delta, cost, io->pzb[p],
                                            io->pzb[p + 1] - io->pzb[p]);
                if (rc) return rc;
                KCS_CUDA_OK(c, cudaEventRecord(io->ev_lm[p], c->stream));
            }
            continue;
        }
        int rc = kcs_launch_lm_step(c, x, x_inner, Tp, tin, first ? 0 : 1, tout, last ? 0 : 1, lin, lout, gamma, delta,
                                    last ? cost : nullptr);
        if (rc) return rc;
    }
    return KCS_OK;
}

int kcs_set_fit_options(kcs_ctx *c, const kcs_fit_options *opt) {
    if (!c) return KCS_ERR_NULL;
    static const kcs_fit_options defaults = {nullptr, 6, nullptr, 0, nullptr, nullptr};
    if (!opt) opt = &defaults;
    if (opt->neighbourhood != 6 && opt->neighbourhood != 10) return fail(c, KCS_ERR_SHAPE, "kcs_set_fit_options: neighbourhood must be 6 or 10");
    const int T = c->cfg.n_frames;
    for (int m = 0; m < T; ++m)
        if (opt->frame_weights && !(opt->frame_weights[m] >= 0.0)) return fail(c, KCS_ERR_SHAPE, "kcs_set_fit_options: negative frame weight");
    for (int p = 0; p < 4; ++p)
        if (opt->delta4 && !(opt->delta4[p] >= 0.0)) return fail(c, KCS_ERR_SHAPE, "kcs_set_fit_options: negative delta");
    if ((opt->box_lo == nullptr) != (opt->box_hi == nullptr)) return fail(c, KCS_ERR_NULL, "kcs_set_fit_options: box_lo and box_hi go together");
    for (int p = 0; p < 4; ++p)
        if (opt->box_lo && !(opt->box_lo[p] <= opt->box_hi[p])) return fail(c, KCS_ERR_SHAPE, "kcs_set_fit_options: box_lo > box_hi");
    c->opt_gen++;
    c->weighted = false;
    for (int m = 0; m < T; ++m) {
        c->h_frames[m].w = opt->frame_weights ? opt->frame_weights[m] : 1.0;
        if (c->h_frames[m].w != 1.0) c->weighted = true;
    }
    KCS_CUDA_OK(c, cudaStreamSynchronize(c->stream));  // kernels in flight still read the old table
    KCS_CUDA_OK(c, cudaMemcpy(c->d_frames, c->h_frames.data(), sizeof(KFrame) * T, cudaMemcpyHostToDevice));
    c->nbr_mode = opt->neighbourhood;
    c->has_delta4 = opt->delta4 != nullptr;
    for (int p = 0; p < 4; ++p) c->delta4[p] = opt->delta4 ? opt->delta4[p] : 0.0;
    c->prior_curv = opt->prior_curvature != 0;
    c->custom_box = opt->box_lo != nullptr;
    const double lo[4] = {0.0, 1e-4, 0.0, 0.0}, hi[4] = {2.0, 2.0, 1.0, 1.0};  // Q16
    for (int p = 0; p < 4; ++p) {
        c->box_lo[p] = opt->box_lo ? opt->box_lo[p] : lo[p];
        c->box_hi[p] = opt->box_hi ? opt->box_hi[p] : hi[p];
    }
    return KCS_OK;
}

int kcs_map_lm(kcs_ctx *c, const float *x, float *theta, float *lambda, float gamma, float delta, int n_steps, float *cost) {
    if (!c) return KCS_ERR_NULL;
    if (!x || !theta || !lambda) return fail(c, KCS_ERR_NULL, "kcs_map_lm: NULL buffer");
    if (n_steps < 0 || !(delta >= 0.f) || !(gamma >= 0.f)) return fail(c, KCS_ERR_SHAPE, "kcs_map_lm: negative n_steps/gamma/delta");
    return lm_steps(c, x, 0, 0, theta, lambda, gamma, delta, n_steps, cost);
}

// F <- K(theta^{n-1}), held fixed during the pass ("one step late").  Only the OSL update needs F, so the evaluator
// runs on a second stream, forked from everything enqueued so far and joined before the first back-projection.
static int start_kinetic(kcs_ctx *c, const float *theta, int Tp) {
    if (!c->aux_stream) {
        KCS_CUDA_OK(c, cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    }
    cudaStream_t main_stream = c->stream;
    KCS_CUDA_OK(c, cudaEventRecord(c->ev_fork, main_stream));
    KCS_CUDA_OK(c, cudaStreamWaitEvent(c->aux_stream, c->ev_fork, 0));
    c->stream = c->aux_stream;
    const int rc = kcs_launch_kinetic(c, theta, c->Fi, nullptr, 1, Tp);
    c->stream = main_stream;
    if (rc) return rc;
    KCS_CUDA_OK(c, cudaEventRecord(c->ev_join, c->aux_stream));
    return KCS_OK;
}

// The z chunks of the host-buffer pipeline.  Nothing can run before the first chunk has arrived, and the last chunk's x
// leaves behind MAP-LM anyway: the LEAD chunk is the smallest that fills the GPU once (148 SMs x 6 forward CTAs of 128
// ray lanes), each following chunk is twice the one before (the OS pass of a slice takes about twice its copy), up to a
// quarter of the volume (>= 16 slices); a remainder of less than half a chunk joins the last one.
static void plan_chunks(const kcs_ctx *c, HostIO &io) {
    const KGeom &g = c->g;
    const double lanes_per_slice = (double)(g.A / g.S) * g.B * (round_up4(c->cfg.n_frames) / 4);
    int s = (int)std::ceil(148.0 * 6 * 128 / lanes_per_slice);
    if (s < 1) s = 1;
    const int cap = (g.nz + 3) / 4 > 16 ? (g.nz + 3) / 4 : 16;
    if (s > cap) s = cap;
    int k = 0, z = 0;
    io.zb[0] = 0;
    while (z < g.nz) {
        int take = s < g.nz - z ? s : g.nz - z;
        if (k == KCS_MAX_CHUNKS - 1 || g.nz - z - take < (take + 1) / 2) take = g.nz - z;
        z += take;
        io.zb[++k] = z;
        s = 2 * s < cap ? 2 * s : cap;
    }
    io.nchunk = k;
}

// The ICM loop.  y, x: DEVICE buffers (the caller's, or the staging buffers of kcs_icm_run_host when io != NULL).
// The OS pass runs chunk by chunk in z (direct planes are independent, so the result does not depend on the chunking);
// with io, chunk k's inputs are awaited just before its first kernel and its final x is handed to the copy-out stream
// right after its last OSL update of the last iteration.
static int icm_run_impl(kcs_ctx *c, const float *y, const float *r, int r_mode, float scale, float *x, float *theta,
                        float *lambda, float beta_first, float beta, float gamma, float delta, int n_lm, int n_iter,
                        HostIO *io) {
    if (!c) return KCS_ERR_NULL;
    if (!y || !r || !x || !theta || !lambda) return fail(c, KCS_ERR_NULL, "kcs_icm: NULL buffer");
    if (r_mode != KCS_R_PER_FRAME && r_mode != KCS_R_FULL) return fail(c, KCS_ERR_SHAPE, "kcs_icm: unknown r_mode");
    if (n_lm < 0 || n_iter < 0 || !(scale > 0.f)) return fail(c, KCS_ERR_SHAPE, "kcs_icm: bad n_lm / n_iter / scale");
    const KGeom &g = c->g;
    const int T = c->cfg.n_frames, Tp = round_up4(T);
    // Two LANES (the context's stream and a second one) carry the OS pass of alternate z chunks.  Direct planes are
    // independent, and while one chunk's kernel drains its last CTAs the other chunk's kernel fills the SMs (every launch
    // ends in a tail of ~0.1 ms, 42 times per chunk and iteration).  Host-buffer mode: the chunks of the copy pipeline.
    // Device-resident call: the volume in two halves -- C2 0.85 -> 0.74 ms (inside its CUDA graph), C3 8.17 -> 7.48 ms,
    // C4 131.8 -> 130.6 ms per iteration; more chunks do not pay (C3: 3 / 4 / 6 / 8 chunks 7.99 / 7.43 / 7.48 / 8.11 ms).
    // One lane for volumes too small to split and while per-kernel timing is on: its events must bracket kernels that
    // have the GPU to themselves.  The result does not depend on the split, bit for bit.
    const bool res2 = !io && !c->prof_on && (double)c->n_vox * T >= 1.0e6 && g.nz >= 8;
    const bool two = (io != nullptr && io->nchunk >= 2 && !c->prof_on) || res2;
    const int whole[3] = {0, res2 ? g.nz / 2 : g.nz, g.nz};
    const int nchunk = io ? io->nchunk : (res2 ? 2 : 1);
    const int *zb = io ? io->zb : whole;
    const int nlane = two ? 2 : 1;
    if (two && !c->os_stream) {
        KCS_CUDA_OK(c, cudaStreamCreateWithFlags(&c->os_stream, cudaStreamNonBlocking));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_os_fork, cudaEventDisableTiming));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_os_join, cudaEventDisableTiming));
    }
    struct StreamRestore {  // the launchers enqueue on c->stream: it is switched per chunk and put back on every exit
        kcs_ctx *c; cudaStream_t s;
        ~StreamRestore() { c->stream = s; }
    } restore{c, c->stream};
    cudaStream_t lanes[2] = {c->stream, c->os_stream};
    int rc;
    // beside the packing and the first forward projection; host-buffer mode: theta arrives chunk by chunk, the first
    // iteration's model curve is evaluated per chunk on the chunk's lane
    if (n_iter > 0 && !io && (rc = start_kinetic(c, theta, Tp))) return rc;
    if ((rc = ensure_border(c, Tp))) return rc;
    if (r_mode == KCS_R_PER_FRAME) {
        KCS_CUDA_OK(c, cudaMemsetAsync(c->r_pad, 0, KCS_MAX_FRAMES * sizeof(float), c->stream));
        KCS_CUDA_OK(c, cudaMemcpyAsync(c->r_pad, r, T * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    } else {
        if (!c->ri) {
            if (dalloc(c, &c->ri, c->n_ray_all * Tp) != cudaSuccess) {
                cudaGetLastError();
                return fail(c, KCS_ERR_ALLOC, "kcs_icm: cannot allocate the packed randoms sinogram");
            }
        }
        if ((rc = pack_sino(c, r, T, c->ri, Tp, g.A))) return rc;
    }
    if (n_iter == 0 || !io) {  // device-resident call: pack everything up front (one chunk)
        if ((rc = pack_image(c, x, T, c->xi, Tp))) return rc;
        if ((rc = pack_sino(c, y, T, c->yi, Tp, g.A))) return rc;
    }
    for (int it = 0; it < n_iter; ++it) {
        const float b = it == 0 ? beta_first : beta;
        const bool last = it == n_iter - 1;
        if (it > 0 && (rc = start_kinetic(c, theta, Tp))) return rc;
        if (two) {  // lane 1 starts behind everything enqueued so far (packing, the previous iteration's MAP-LM)
            KCS_CUDA_OK(c, cudaEventRecord(c->ev_os_fork, lanes[0]));
            KCS_CUDA_OK(c, cudaStreamWaitEvent(lanes[1], c->ev_os_fork, 0));
        }
        bool has_F[2] = {false, false};
        for (int k = 0; k < nchunk; ++k) {
            const int z0 = zb[k], nzc = zb[k + 1] - zb[k];
            if (nzc == 0) continue;
            const int lane = k % nlane;
            c->stream = lanes[lane];
            if (io && it == 0) {  // this chunk's x, y and theta have been copied to the staging buffers
                KCS_CUDA_OK(c, cudaStreamWaitEvent(c->stream, c->ev_in[k], 0));
                if ((rc = pack_image(c, x, T, c->xi, Tp, z0, nzc))) return rc;
                if ((rc = pack_sino(c, y, T, c->yi, Tp, g.A, z0, nzc))) return rc;
                if ((rc = kcs_launch_kinetic(c, theta, c->Fi, nullptr, 1, Tp, z0, nzc))) return rc;
            }
            for (int s = 0; s < g.S; ++s) {  // Q5: subsets in order 0..S-1
                // after the first OSL update of this call x is zero outside the mask: rays are clipped to the FOV circle
                if ((rc = kcs_launch_forward(c, Tp, s, 1, scale, r_mode, (it > 0 || s > 0) ? 1 : 0, z0, nzc))) return rc;
                if (!has_F[lane] && !(io && it == 0)) {  // the model curve (second stream) is needed from the first OSL update on
                    KCS_CUDA_OK(c, cudaStreamWaitEvent(c->stream, c->ev_join, 0));
                    has_F[lane] = true;
                }
                if ((rc = kcs_launch_back(c, Tp, s, 1, nullptr, scale, b, z0, nzc))) return rc;
            }
            if (io && last) {  // this chunk's activity is final: unpack it and let the copy-out stream take it
                if ((rc = unpack_image(c, c->xi, Tp, x, T, z0, nzc))) return rc;
                KCS_CUDA_OK(c, cudaEventRecord(c->ev_out[k], c->stream));
            }
        }
        c->stream = lanes[0];
        if (two) {
            KCS_CUDA_OK(c, cudaEventRecord(c->ev_os_join, lanes[1]));
            KCS_CUDA_OK(c, cudaStreamWaitEvent(lanes[0], c->ev_os_join, 0));
        }
        if (last && !io) {  // the activity is final after the last OS pass; MAP-LM only reads it: unpack beside the fit
            cudaStream_t main_stream = c->stream;
            KCS_CUDA_OK(c, cudaEventRecord(c->ev_fork, main_stream));
            KCS_CUDA_OK(c, cudaStreamWaitEvent(c->aux_stream, c->ev_fork, 0));
            c->stream = c->aux_stream;
            rc = unpack_image(c, c->xi, Tp, x, T);
            c->stream = main_stream;
            if (rc) return rc;
            KCS_CUDA_OK(c, cudaEventRecord(c->ev_join, c->aux_stream));
        }
        if (io && it == 0) KCS_CUDA_OK(c, cudaStreamWaitEvent(c->stream, io->ev_lam, 0));
        if ((rc = lm_steps(c, c->xi, 1, Tp, theta, lambda, gamma, delta, n_lm, nullptr, last ? io : nullptr))) return rc;
        if (last && !io) KCS_CUDA_OK(c, cudaStreamWaitEvent(c->stream, c->ev_join, 0));
    }
    if (n_iter == 0) {
        if ((rc = unpack_image(c, c->xi, Tp, x, T))) return rc;
    }
    return KCS_OK;
}

// S:7-H6.  A small problem's ICM iteration is ~20 kernels of a few microseconds each: launch-bound.  The first
// kcs_icm_run with a given set of arguments is CAPTURED into a CUDA graph (the second-stream fork / join included) and
// launched; later calls with the same arguments replay it with one cudaGraphLaunch.  The graph bakes in pointers and
// scalars only -- buffer CONTENTS are read at replay time -- and is dropped when an option it depends on changes.
// Not used while per-kernel profiling is on, when the caller's stream is itself being captured, or for volumes that
// are not launch-bound.
static bool graph_eligible(kcs_ctx *c, int n_iter) {
    if (!c->use_graphs || c->prof_on || n_iter <= 0 || n_iter > 16) return false;
    if ((double)c->n_vox * c->cfg.n_frames > 4.0e6) return false;  // C1, C2-sized; C3 and C4 keep the GPU busy per launch
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(c->stream, &st) != cudaSuccess || st != cudaStreamCaptureStatusNone) { cudaGetLastError(); return false; }
    return true;
}

int kcs_icm_run(kcs_ctx *c, const float *y, const float *r, int r_mode, float scale, float *x, float *theta, float *lambda,
                float beta_first, float beta, float gamma, float delta, int n_lm, int n_iter) {
    if (!c) return KCS_ERR_NULL;
    if (!y || !r || !x || !theta || !lambda || (r_mode != KCS_R_PER_FRAME && r_mode != KCS_R_FULL) || n_lm < 0 || !(scale > 0.f) ||
        !graph_eligible(c, n_iter))
        return icm_run_impl(c, y, r, r_mode, scale, x, theta, lambda, beta_first, beta, gamma, delta, n_lm, n_iter, nullptr);
    for (size_t q = 0; q < c->graphs.size(); ++q) {
        const KGraphEntry &ge = c->graphs[q];
        if (ge.y == y && ge.r == r && ge.x == x && ge.theta == theta && ge.lambda == lambda && ge.r_mode == r_mode &&
            ge.n_lm == n_lm && ge.n_iter == n_iter && ge.scale == scale && ge.beta_first == beta_first && ge.beta == beta &&
            ge.gamma == gamma && ge.delta == delta && ge.stream == c->stream && ge.gen == c->opt_gen) {
            // an intervening call with another frame count may have left xi with another layout: the border must be valid
            int rc = ensure_border(c, round_up4(c->cfg.n_frames));
            if (rc) return rc;
            KCS_CUDA_OK(c, cudaGraphLaunch(ge.exec, c->stream));
            c->launches += ge.launches;
            c->graph_replays++;
            return KCS_OK;
        }
    }
    // everything that may not happen during capture happens now: allocations, stream / event creation, the border memset
    const int Tp = round_up4(c->cfg.n_frames);
    int rc = ensure_border(c, Tp);
    if (rc) return rc;
    if (r_mode == KCS_R_FULL && !c->ri && dalloc(c, &c->ri, c->n_ray_all * Tp) != cudaSuccess) {
        cudaGetLastError();
        return fail(c, KCS_ERR_ALLOC, "kcs_icm: cannot allocate the packed randoms sinogram");
    }
    if (!c->aux_stream) {
        KCS_CUDA_OK(c, cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    }
    const long long n0 = c->launches;
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        return icm_run_impl(c, y, r, r_mode, scale, x, theta, lambda, beta_first, beta, gamma, delta, n_lm, n_iter, nullptr);
    }
    rc = icm_run_impl(c, y, r, r_mode, scale, x, theta, lambda, beta_first, beta, gamma, delta, n_lm, n_iter, nullptr);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (rc != KCS_OK || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        if (rc != KCS_OK) return rc;
        c->launches = n0;  // capture failed: run the call directly
        return icm_run_impl(c, y, r, r_mode, scale, x, theta, lambda, beta_first, beta, gamma, delta, n_lm, n_iter, nullptr);
    }
    KGraphEntry ge{y, r, x, theta, lambda, r_mode, n_lm, n_iter, scale, beta_first, beta, gamma, delta, c->stream, c->opt_gen,
                   c->launches - n0, nullptr};
    e = cudaGraphInstantiate(&ge.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
        cudaGetLastError();
        c->launches = n0;
        return icm_run_impl(c, y, r, r_mode, scale, x, theta, lambda, beta_first, beta, gamma, delta, n_lm, n_iter, nullptr);
    }
    // keep the graphs of the current option generation only, at most 8 of them
    for (size_t q = 0; q < c->graphs.size();) {
        if (c->graphs[q].gen != c->opt_gen || c->graphs.size() >= 8) { cudaGraphExecDestroy(c->graphs[q].exec); c->graphs.erase(c->graphs.begin() + q); }
        else ++q;
    }
    c->graphs.push_back(ge);
    KCS_CUDA_OK(c, cudaGraphLaunch(ge.exec, c->stream));
    return KCS_OK;
}

int kcs_icm_iteration(kcs_ctx *c, const float *y, const float *r, int r_mode, float scale, float *x, float *theta,
                      float *lambda, float beta, float gamma, float delta, int n_lm) {
    return kcs_icm_run(c, y, r, r_mode, scale, x, theta, lambda, beta, beta, gamma, delta, n_lm, 1);
}

int kcs_icm_run_host(kcs_ctx *c, const float *y, const float *r, int r_mode, float scale, float *x, float *theta,
                     float *lambda, float beta_first, float beta, float gamma, float delta, int n_lm, int n_iter) {
    if (!c) return KCS_ERR_NULL;
    if (!y || !r || !x || !theta || !lambda) return fail(c, KCS_ERR_NULL, "kcs_icm_run_host: NULL buffer");
    if (r_mode != KCS_R_PER_FRAME && r_mode != KCS_R_FULL) return fail(c, KCS_ERR_SHAPE, "kcs_icm_run_host: unknown r_mode");
    const KGeom &g = c->g;
    const int T = c->cfg.n_frames;
    const size_t ny_ = (size_t)T * c->n_ray_all, nx_ = (size_t)T * c->n_vox;
    const size_t nr = r_mode == KCS_R_PER_FRAME ? (size_t)T : ny_;
    cudaError_t e = cudaSuccess;
    if (!c->st_y) {
        if (e == cudaSuccess) e = dalloc(c, &c->st_y, ny_);
        if (e == cudaSuccess) e = dalloc(c, &c->st_x, nx_);
        if (e == cudaSuccess) e = dalloc(c, &c->st_theta, 4 * c->n_vox);
        if (e == cudaSuccess) e = dalloc(c, &c->st_lambda, c->n_vox);
    }
    if (e == cudaSuccess && c->st_r_elems < nr) {
        if (c->st_r) cudaFree(c->st_r);
        c->st_r = nullptr;
        e = dalloc(c, &c->st_r, nr);
        c->st_r_elems = e == cudaSuccess ? nr : 0;
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, KCS_ERR_ALLOC, std::string("kcs_icm_run_host: ") + cudaGetErrorString(e));
    }
    HostIO io{};
    io.hy = y; io.hx = x;
    plan_chunks(c, io);
    if (!c->in_stream) {
        KCS_CUDA_OK(c, cudaStreamCreateWithFlags(&c->in_stream, cudaStreamNonBlocking));
        KCS_CUDA_OK(c, cudaStreamCreateWithFlags(&c->out_stream, cudaStreamNonBlocking));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_small, cudaEventDisableTiming));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_lam, cudaEventDisableTiming));
    }
    io.ev_lam = c->ev_lam;
    while ((int)c->ev_lm.size() < KCS_LM_PIECES) {
        cudaEvent_t a = nullptr;
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        c->ev_lm.push_back(a);
    }
    for (int p = 0; p < KCS_LM_PIECES; ++p) io.ev_lm[p] = c->ev_lm[p];
    while ((int)c->ev_in.size() < io.nchunk) {
        cudaEvent_t a = nullptr, b = nullptr;
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        KCS_CUDA_OK(c, cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
        c->ev_in.push_back(a);
        c->ev_out.push_back(b);
    }
    cudaStream_t st = c->stream, in = c->in_stream, out = c->out_stream;
    // the copy-in stream starts behind whatever the caller has enqueued on the context's stream (the staging buffers
    // may still be in use by a previous call)
    KCS_CUDA_OK(c, cudaEventRecord(c->ev_small, st));
    KCS_CUDA_OK(c, cudaStreamWaitEvent(in, c->ev_small, 0));
    // order on the copy-in stream: r (the first ratio needs it), the chunks, lambda last (only MAP-LM reads it)
    KCS_CUDA_OK(c, cudaMemcpyAsync(c->st_r, r, nr * sizeof(float), cudaMemcpyHostToDevice, in));
    KCS_CUDA_OK(c, cudaEventRecord(c->ev_small, in));
    for (int k = 0; k < io.nchunk; ++k) {  // x, y and theta of chunk k: T resp. 4 strided pieces each (one 2-D copy)
        const int z0 = io.zb[k], nzc = io.zb[k + 1] - io.zb[k];
        if (nzc > 0) {
            const size_t v2 = (size_t)g.ny * g.nx, r2 = (size_t)g.A * g.B;
            KCS_CUDA_OK(c, cudaMemcpy2DAsync(c->st_theta + z0 * v2, c->n_vox * sizeof(float), theta + z0 * v2, c->n_vox * sizeof(float),
                                             nzc * v2 * sizeof(float), 4, cudaMemcpyHostToDevice, in));
            KCS_CUDA_OK(c, cudaMemcpy2DAsync(c->st_x + z0 * v2, c->n_vox * sizeof(float), x + z0 * v2, c->n_vox * sizeof(float),
                                             nzc * v2 * sizeof(float), T, cudaMemcpyHostToDevice, in));
            KCS_CUDA_OK(c, cudaMemcpy2DAsync(c->st_y + z0 * r2, c->n_ray_all * sizeof(float), y + z0 * r2,
                                             c->n_ray_all * sizeof(float), nzc * r2 * sizeof(float), T, cudaMemcpyHostToDevice, in));
        }
        KCS_CUDA_OK(c, cudaEventRecord(c->ev_in[k], in));
    }
    KCS_CUDA_OK(c, cudaMemcpyAsync(c->st_lambda, lambda, c->n_vox * sizeof(float), cudaMemcpyHostToDevice, in));
    KCS_CUDA_OK(c, cudaEventRecord(c->ev_lam, in));
    KCS_CUDA_OK(c, cudaStreamWaitEvent(st, c->ev_small, 0));
    if (n_iter <= 0) {  // nothing to overlap: wait for every chunk, the loop below only unpacks
        for (int k = 0; k < io.nchunk; ++k) KCS_CUDA_OK(c, cudaStreamWaitEvent(st, c->ev_in[k], 0));
        KCS_CUDA_OK(c, cudaStreamWaitEvent(st, c->ev_lam, 0));
    }
    int rc = icm_run_impl(c, c->st_y, c->st_r, r_mode, scale, c->st_x, c->st_theta, c->st_lambda, beta_first, beta, gamma, delta,
                          n_lm, n_iter, n_iter > 0 ? &io : nullptr);
    if (rc) return rc;
    if (n_iter > 0) {
        for (int k = 0; k < io.nchunk; ++k) {  // x of chunk k goes back while later chunks and the last MAP-LM still run
            const int z0 = io.zb[k], nzc = io.zb[k + 1] - io.zb[k];
            if (nzc == 0) continue;
            const size_t v2 = (size_t)g.ny * g.nx;
            KCS_CUDA_OK(c, cudaStreamWaitEvent(out, c->ev_out[k], 0));
            KCS_CUDA_OK(c, cudaMemcpy2DAsync(x + z0 * v2, c->n_vox * sizeof(float), c->st_x + z0 * v2, c->n_vox * sizeof(float),
                                             nzc * v2 * sizeof(float), T, cudaMemcpyDeviceToHost, out));
        }
    } else {
        KCS_CUDA_OK(c, cudaMemcpyAsync(x, c->st_x, nx_ * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    if (io.n_piece > 0) {  // theta and lambda of a z piece leave while the last MAP-LM step fits the next piece
        const size_t v2 = (size_t)g.ny * g.nx;
        for (int p = 0; p < io.n_piece; ++p) {
            const size_t z0 = (size_t)io.pzb[p], nzp = (size_t)(io.pzb[p + 1] - io.pzb[p]);
            KCS_CUDA_OK(c, cudaStreamWaitEvent(out, io.ev_lm[p], 0));
            KCS_CUDA_OK(c, cudaMemcpy2DAsync(theta + z0 * v2, c->n_vox * sizeof(float), c->st_theta + z0 * v2, c->n_vox * sizeof(float),
                                             nzp * v2 * sizeof(float), 4, cudaMemcpyDeviceToHost, out));
            KCS_CUDA_OK(c, cudaMemcpyAsync(lambda + z0 * v2, c->st_lambda + z0 * v2, nzp * v2 * sizeof(float), cudaMemcpyDeviceToHost, out));
        }
    } else {
        KCS_CUDA_OK(c, cudaMemcpyAsync(theta, c->st_theta, 4 * c->n_vox * sizeof(float), cudaMemcpyDeviceToHost, st));
        KCS_CUDA_OK(c, cudaMemcpyAsync(lambda, c->st_lambda, c->n_vox * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    KCS_CUDA_OK(c, cudaStreamSynchronize(st));
    KCS_CUDA_OK(c, cudaStreamSynchronize(out));
    KCS_CUDA_OK(c, cudaStreamSynchronize(in));
    return KCS_OK;
}

}  // extern "C"
