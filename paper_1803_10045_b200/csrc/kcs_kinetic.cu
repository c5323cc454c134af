// kcs_kinetic.cu -- frame-integrated 2-tissue irreversible FDG model (K1-K6) and the batched per-voxel MAP-LM
// solver (L1-L3).  sm_100a.
//
// Cited passages: P:85-89 (analytic time integrals and derivatives), P:91-114 (eq. 4-7), BJ configs[0](1)-(3).
//
// Precision: the closed-form W_m(a) = int_frame (e^{-a.} conv Cp) cancels catastrophically in fp32
// (1.5e-3 relative error at a = 0.19, >100 % near a = lambda_i), so the per-voxel model, the 4x4 normal
// equations and the accept/reject test run in fp64 registers; global memory traffic is fp32.
//
// Formulation.  With c_i = a - l_i, E0(t) = int_0^t e^{-au} du, E1(t) = int_0^t u e^{-au} du (both advanced from
// frame to frame by the positive recurrences E0(t+d) = E0(t) + e^{-at} E0(d), E1(t+d) = E1(t) + e^{-at}(t E0(d) + E1(d)),
// so one expm1 per distinct frame duration suffices) and host tables P_n(l_i; t) = int_0^t u^n e^{-l_i u} du:
//     D_i = (P0(l_i;t) - E0)/c_i                 T_0 = (P1(l_0;t) - D_0)/c_0
//     G_a(t) = int_0^t (e^{-a.} conv Cp) = sum_i alpha_i D_i + beta_0 T_0
//     dD_i/da = (E1 - D_i)/c_i                   dT_0/da = -(dD_0/da + T_0)/c_0
// and for |c_i| < 1e-4 (i = 1, 2; l_0 = 4.134 is outside the parameter box) the Taylor expansion about a = l_i:
//     D_i = P1 - P2 c/2 + P3 c^2/6 - P4 c^3/24,  dD_i/da = -P2/2 + P3 c/3 - P4 c^2/8.
#include "kcs_internal.cuh"

#define LAUNCH_CHECK(c)                                                     \
    do {                                                                    \
        (c)->launches++;                                                    \
        cudaError_t e__ = cudaGetLastError();                               \
        if (e__ != cudaSuccess) {                                           \
            (c)->err = std::string("kernel launch: ") + cudaGetErrorString(e__); \
            return KCS_ERR_CUDA;                                            \
        }                                                                   \
    } while (0)

namespace {

// Options of the fit handed to k_lm_step by value (kcs_set_fit_options; the default kernel reads delta[0] only).
struct LmOpt {
    double delta[4];      // Huber threshold per parameter map
    double lo[4], hi[4];  // parameter box; lo == hi fixes a parameter
    int nq;               // neighbours: 6 or 10
    int curv;             // Huber curvature in the LM matrix
    int fixmask;          // bit p: parameter p is fixed
};

// E1(a; t) = int_0^t u e^{-a u} du, given z = a t and em1 = expm1(-z).
__device__ __forceinline__ double E1_of(double a, double t, double z, double em1) {
    if (z < 0.5) {
        // t^2 sum_{n>=0} (-z)^n / (n! (n+2)), Horner with c_n = 1/(n! (n+2)); 15 terms: 0.5^15/15!/17 < 2e-18
        const double w = -z;
        double s = 1.0 / (87178291200.0 * 16.0);                 // n = 14
        s = fma(s, w, 1.0 / (6227020800.0 * 15.0));              // 13
        s = fma(s, w, 1.0 / (479001600.0 * 14.0));               // 12
        s = fma(s, w, 1.0 / (39916800.0 * 13.0));                // 11
        s = fma(s, w, 1.0 / (3628800.0 * 12.0));                 // 10
        s = fma(s, w, 1.0 / (362880.0 * 11.0));                  // 9
        s = fma(s, w, 1.0 / (40320.0 * 10.0));                   // 8
        s = fma(s, w, 1.0 / (5040.0 * 9.0));                     // 7
        s = fma(s, w, 1.0 / (720.0 * 8.0));                      // 6
        s = fma(s, w, 1.0 / (120.0 * 7.0));                      // 5
        s = fma(s, w, 1.0 / (24.0 * 6.0));                       // 4
        s = fma(s, w, 1.0 / (6.0 * 5.0));                        // 3
        s = fma(s, w, 1.0 / (2.0 * 4.0));                        // 2
        s = fma(s, w, 1.0 / 3.0);                                // 1
        s = fma(s, w, 0.5);                                      // 0
        return t * t * s;
    }
    return (-em1 - z * (1.0 + em1)) / (a * a);
}

struct VoxRate {  // per-voxel, rate-dependent scalars
    double a, ic[3], c[3];
    bool tay[3];
};

__device__ __forceinline__ void rate_setup(const KKin &kin, double a, VoxRate &r) {
    r.a = a;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        r.c[i] = a - kin.lam[i];
        r.tay[i] = (i > 0) && (fabs(r.c[i]) < 1e-4);
        r.ic[i] = r.tay[i] ? 0.0 : 1.0 / r.c[i];
    }
}

// G_a(t) and dG_a/da at a boundary, given E0 = P0(a;t), E1 = P1(a;t).
__device__ __forceinline__ void G_at(const KKin &kin, const KBoundary &b, const VoxRate &r, double E0, double E1,
                                     double &G, double &dG) {
    const double D0 = (b.P0[0] - E0) * r.ic[0];
    const double T0 = (b.P1_0 - D0) * r.ic[0];
    const double dD0 = (E1 - D0) * r.ic[0];
    const double dT0 = -(dD0 + T0) * r.ic[0];
    G = kin.alpha[0] * D0 + kin.beta0 * T0;
    dG = kin.alpha[0] * dD0 + kin.beta0 * dT0;
#pragma unroll
    for (int i = 1; i < 3; ++i) {
        double D, dD;
        if (!r.tay[i]) {
            D = (b.P0[i] - E0) * r.ic[i];
            dD = (E1 - D) * r.ic[i];
        } else {
            const double c = r.c[i];
            const double *P = b.Pn[i - 1];
            D = P[0] + c * (-0.5 * P[1] + c * (P[2] * (1.0 / 6.0) - c * P[3] * (1.0 / 24.0)));
            dD = -0.5 * P[1] + c * (P[2] * (1.0 / 3.0) - c * P[3] * 0.125);
        }
        G += kin.alpha[i] * D;
        dG += kin.alpha[i] * dD;
    }
}

// Streams over the frames of one voxel and hands (m, F_m, dF/dK1, dF/dk2, dF/dk3, dF/dvB) to `sink`.
// K2, K3, K6.  fr = frame tables (shared memory).
template <bool JAC, class Sink>
__device__ __forceinline__ void tac_stream(const KKin &kin, const KFrame *fr, double K1, double k2, double k3, double vB,
                                           Sink &&sink) {
    const double a = k2 + k3;
    const int T = kin.T;
    if (!(a > 0.0)) {  // k2 = k3 = 0: the bracket of K2 reduces to K1 (1 conv Cp)
        for (int m = 0; m < T; ++m) {
            const double W0 = fr[m].W0, dI = fr[m].dICp;
            sink(m, vB * dI + (1.0 - vB) * K1 * W0, (1.0 - vB) * W0, 0.0, 0.0, dI - K1 * W0);
        }
        return;
    }
    VoxRate r;
    rate_setup(kin, a, r);
    const double ia = 1.0 / a;
    const double B1 = K1 * k2 * ia, B2 = K1 * k3 * ia;
    const double omv = 1.0 - vB;
    const double k2a = k2 * ia, k3a = k3 * ia;
    const double c23 = K1 * k3 * ia * ia, c32 = K1 * k2 * ia * ia;
    double e = 1.0, E0 = 0.0, E1 = 0.0, Gs = 0.0, dGs = 0.0;  // state at the current frame start
    double ed = 1.0, E0d = 0.0, E1d = 0.0;                    // per-duration scalars
    for (int m = 0; m < T; ++m) {
        const KFrame &f = fr[m];
        if (!f.contiguous) {
            const double ts = f.b[0].t;
            if (ts > 0.0) {
                const double z = a * ts, em1 = expm1(-z);
                e = 1.0 + em1;
                E0 = -em1 * ia;
                E1 = E1_of(a, ts, z, em1);
                G_at(kin, f.b[0], r, E0, E1, Gs, dGs);
            } else {
                e = 1.0; E0 = 0.0; E1 = 0.0; Gs = 0.0; dGs = 0.0;
            }
        }
        if (f.new_dt) {
            const double z = a * f.dt, em1 = expm1(-z);
            ed = 1.0 + em1;
            E0d = -em1 * ia;
            E1d = E1_of(a, f.dt, z, em1);
        }
        const double ts = f.b[0].t;
        const double E1e = E1 + e * (ts * E0d + E1d);
        const double E0e = E0 + e * E0d;
        const double ee = e * ed;
        double Ge, dGe;
        G_at(kin, f.b[1], r, E0e, E1e, Ge, dGe);
        const double W = Ge - Gs;
        const double tissue = B1 * W + B2 * f.W0;
        const double F = vB * f.dICp + omv * tissue;
        if (JAC) {
            const double dW = dGe - dGs;
            sink(m, F, omv * (k2a * W + k3a * f.W0), omv * (c23 * (W - f.W0) + B1 * dW),
                 omv * (c32 * (f.W0 - W) + B1 * dW), f.dICp - tissue);
        } else {
            sink(m, F, 0.0, 0.0, 0.0, 0.0);
        }
        e = ee; E0 = E0e; E1 = E1e; Gs = Ge; dGs = dGe;
    }
}

__device__ __forceinline__ void load_frames(const KKin &kin, KFrame *sh) {
    const int n = kin.T * (int)(sizeof(KFrame) / sizeof(double));
    const double *src = reinterpret_cast<const double *>(kin.frames);
    double *dst = reinterpret_cast<double *>(sh);
    for (int q = threadIdx.x; q < n; q += blockDim.x) dst[q] = src[q];
    __syncthreads();
}

struct XAddr {  // where voxel v's frame m lives: base + m * fstride
    size_t base;
    size_t fstride;
};
__device__ __forceinline__ XAddr x_addr(const KGeom &g, size_t nvox, long long v, int inner, int Tp) {
    XAddr r;
    if (!inner) {
        r.base = (size_t)v;
        r.fstride = nvox;
    } else {
        const int v2 = g.nx * g.ny;
        const int z = (int)(v / v2), rem = (int)(v - (long long)z * v2);
        const int j = rem / g.nx, i = rem - j * g.nx;
        r.base = (((size_t)z * g.nyp + (j + KCS_PAD)) * g.nxp + (i + KCS_PAD)) * Tp;
        r.fstride = 1;
    }
    return r;
}

// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_kinetic(KGeom g, KKin kin, const float *__restrict__ theta, float *F, float *J,
                                                 long long nvox, int inner, int Tp) {
    extern __shared__ double sh_raw[];
    KFrame *fr = reinterpret_cast<KFrame *>(sh_raw);
    load_frames(kin, fr);
    const long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    const double K1 = theta[v], k2 = theta[nvox + v], k3 = theta[2 * nvox + v], vB = theta[3 * nvox + v];
    const XAddr xa = x_addr(g, (size_t)nvox, v, inner, Tp);
    const size_t TV = (size_t)kin.T * nvox;
    if (J) {
        tac_stream<true>(kin, fr, K1, k2, k3, vB, [&](int m, double Fm, double j0, double j1, double j2, double j3) {
            F[xa.base + m * xa.fstride] = (float)Fm;
            const size_t o = (size_t)m * nvox + v;
            J[o] = (float)j0; J[TV + o] = (float)j1; J[2 * TV + o] = (float)j2; J[3 * TV + o] = (float)j3;
        });
    } else {
        tac_stream<false>(kin, fr, K1, k2, k3, vB, [&](int m, double Fm, double, double, double, double) {
            F[xa.base + m * xa.fstride] = (float)Fm;
        });
    }
}

// The model curve of the ICM path (a1): in-mask voxels only (the OSL update reads F nowhere else; the rest of Fi keeps the
// zeros it was created with), written to the padded frame-innermost layout four frames at a time (one 16 B store per
// lane instead of four scattered 4 B stores; frames T..Tp-1 are written as 0).
__global__ void __launch_bounds__(128) k_kinetic_inner(KGeom g, KKin kin, const float *__restrict__ theta, float *F, long long nvox,
                                                       const int *__restrict__ vlist, int M2, int Tp, long long t0, long long t1) {
    extern __shared__ double sh_raw[];
    KFrame *fr = reinterpret_cast<KFrame *>(sh_raw);
    load_frames(kin, fr);
    const long long t = t0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;  // [t0, t1): the in-mask voxels of a z range
    if (t >= t1) return;
    const int v2 = g.nx * g.ny;
    const int z = (int)(t / M2), rem = vlist[(int)(t - (long long)z * M2)];
    const long long v = (long long)z * v2 + rem;
    const double K1 = theta[v], k2 = theta[nvox + v], k3 = theta[2 * nvox + v], vB = theta[3 * nvox + v];
    const XAddr xa = x_addr(g, (size_t)nvox, v, 1, Tp);
    float4 *dst = reinterpret_cast<float4 *>(F + xa.base);
    float b0 = 0.f, b1 = 0.f, b2 = 0.f, b3 = 0.f;  // a four-frame shift register (no dynamic register indexing)
    const int T = kin.T;
    tac_stream<false>(kin, fr, K1, k2, k3, vB, [&](int m, double Fm, double, double, double, double) {
        b0 = b1; b1 = b2; b2 = b3; b3 = (float)Fm;
        if (m == T - 1)
            for (int pad = 3 - (m & 3); pad > 0; --pad) { b0 = b1; b1 = b2; b2 = b3; b3 = 0.f; }  // the last, partial group
        if ((m & 3) == 3 || m == T - 1) dst[m >> 2] = make_float4(b0, b1, b2, b3);
    });
    for (int q = (T + 3) / 4; q < Tp / 4; ++q) dst[q] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// ---------------------------------------------------------------------------------------------------------
// MAP-LM step (L1-L3).  One thread = one voxel; everything per-voxel lives in fp64 registers.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double huber(double t, double d) {  // eq. 5 with Q12
    const double at = fabs(t);
    return at <= d ? 0.5 * t * t : d * at - 0.5 * d * d;
}
__device__ __forceinline__ double huber_d(double t, double d) {  // eq. 6 with Q12
    return fmin(fmax(t, -d), d);
}

// Cholesky solve of the 4x4 SPD system M d = g (M given by its lower triangle, row-major packed m[10]).
__device__ __forceinline__ bool chol4(const double m[10], const double g[4], double d[4]) {
    // packed index: (0,0)=0 (1,0)=1 (1,1)=2 (2,0)=3 (2,1)=4 (2,2)=5 (3,0)=6 (3,1)=7 (3,2)=8 (3,3)=9
    double l00, l10, l11, l20, l21, l22, l30, l31, l32, l33, s;
    s = m[0]; if (!(s > 0.0) || !isfinite(s)) return false; l00 = sqrt(s);
    l10 = m[1] / l00;
    s = m[2] - l10 * l10; if (!(s > 0.0) || !isfinite(s)) return false; l11 = sqrt(s);
    l20 = m[3] / l00;
    l21 = (m[4] - l20 * l10) / l11;
    s = m[5] - l20 * l20 - l21 * l21; if (!(s > 0.0) || !isfinite(s)) return false; l22 = sqrt(s);
    l30 = m[6] / l00;
    l31 = (m[7] - l30 * l10) / l11;
    l32 = (m[8] - l30 * l20 - l31 * l21) / l22;
    s = m[9] - l30 * l30 - l31 * l31 - l32 * l32; if (!(s > 0.0) || !isfinite(s)) return false; l33 = sqrt(s);
    const double z0 = g[0] / l00;
    const double z1 = (g[1] - l10 * z0) / l11;
    const double z2 = (g[2] - l20 * z0 - l21 * z1) / l22;
    const double z3 = (g[3] - l30 * z0 - l31 * z1 - l32 * z2) / l33;
    d[3] = z3 / l33;
    d[2] = (z2 - l32 * d[3]) / l22;
    d[1] = (z1 - l21 * d[2] - l31 * d[3]) / l11;
    d[0] = (z0 - l10 * d[1] - l20 * d[2] - l30 * d[3]) / l00;
    return true;
}

// Data part of the normal equations at theta: out[0..9] = J^T J (packed lower triangle), out[10..13] = J^T r,
// out[14] = 1/2 sum r^2.  One (not inlined) copy of the model code serves both evaluations of a step.
// WLS (the OPT kernel): frame weights, and `fixmask` bit p set = parameter p is fixed (its Jacobian column is zero).
template <bool WLS>
__device__ __forceinline__ void lm_eval(KKin kin, const KFrame *fr, const float *__restrict__ x, size_t xbase, size_t xstride,
                                     double K1, double k2, double k3, double vB, int fixmask, double *out) {
    double JtJ[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, gr[4] = {0, 0, 0, 0}, phi = 0.0;
    const double f0 = (fixmask & 1) ? 0.0 : 1.0, f1 = (fixmask & 2) ? 0.0 : 1.0, f2 = (fixmask & 4) ? 0.0 : 1.0, f3 = (fixmask & 8) ? 0.0 : 1.0;
    tac_stream<true>(kin, fr, K1, k2, k3, vB, [&](int m, double Fm, double j0, double j1, double j2, double j3) {
        const double r = (double)x[xbase + m * xstride] - Fm;
        if (WLS) { j0 *= f0; j1 *= f1; j2 *= f2; j3 *= f3; }
        // S8(f)4: frame weights w_m (WLS; compiled out of the default path) -- J^T W J, J^T W r, 1/2 r^T W r
        const double w = WLS ? fr[m].w : 1.0;
        const double w0 = WLS ? w * j0 : j0, w1 = WLS ? w * j1 : j1, w2 = WLS ? w * j2 : j2, w3 = WLS ? w * j3 : j3;
        phi += WLS ? 0.5 * (w * r) * r : 0.5 * r * r;
        JtJ[0] += w0 * j0;
        JtJ[1] += w1 * j0; JtJ[2] += w1 * j1;
        JtJ[3] += w2 * j0; JtJ[4] += w2 * j1; JtJ[5] += w2 * j2;
        JtJ[6] += w3 * j0; JtJ[7] += w3 * j1; JtJ[8] += w3 * j2; JtJ[9] += w3 * j3;
        gr[0] += w0 * r; gr[1] += w1 * r; gr[2] += w2 * r; gr[3] += w3 * r;
    });
#pragma unroll
    for (int q = 0; q < 10; ++q) out[q] = JtJ[q];
#pragma unroll
    for (int q = 0; q < 4; ++q) out[10 + q] = gr[q];
    out[14] = phi;
}

// 5 CTAs of 128 threads per SM (<= 102 registers): measured best of 1..8 on C2 and C4
// TI / TO: storage type of the maps and of lambda on input / output.  Between the steps of one kcs_map_lm call the
// iterate is kept in fp64 ping-pong buffers (TI = TO = double); only the caller's buffers are fp32.
// OPT = false: the hot path of S8(a) (6 neighbours, one delta, unweighted).  OPT = true: the options of kcs_set_fit_options
// (frame weights, nq = 6 or 10 neighbours, one delta per parameter), kept out of the default kernel's registers.
template <class TI, class TO, bool OPT>
#define KCS_LM_TPB 128
#define KCS_LM_MINBLK 5
// One thread per IN-MASK voxel: thread t of the launch fits voxel (z = t / M2, pixel vlist[t % M2]), M2 = in-mask pixels
// of a slice.  Out-of-mask voxels get no thread (they are never read as neighbours and never written).
__global__ void __launch_bounds__(KCS_LM_TPB, KCS_LM_MINBLK) k_lm_step(KGeom g, KKin kin, const float *__restrict__ x, int x_inner, int Tp,
                                                 const TI *__restrict__ th_in, TO *__restrict__ th_out,
                                                 const TI *lam_in, TO *lam_out,  // may alias: each thread touches its own element
                                                 const unsigned char *__restrict__ mask, const int *__restrict__ vlist, int M2,
                                                 long long nvox, double gamma, LmOpt o, float *cost,
                                                 double *__restrict__ st, long long nfit, long long t0, long long t1) {
    constexpr int NQ = OPT ? 10 : 6;
    constexpr bool WLS = OPT;
    // FIRST step of a call (fp32 input): the data part of the normal equations is evaluated at theta.  Later steps read
    // it from `st` [15][nfit], where the previous step left it for the iterate it produced: an accepted trial point was
    // evaluated WITH its Jacobian, a rejected step leaves theta -- and therefore J^T J, J^T r, Phi_data -- unchanged.
    // So a step costs one model + Jacobian evaluation instead of one with and one without.
    constexpr bool FIRST = sizeof(TI) == 4, LAST = sizeof(TO) == 4;
    extern __shared__ double sh_raw[];
    KFrame *fr = reinterpret_cast<KFrame *>(sh_raw);
    load_frames(kin, fr);
    const long long t = t0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;  // [t0, t1): the in-mask voxels of a z range
    if (t >= t1) return;
    const int v2 = g.nx * g.ny;
    const int z = (int)(t / M2), rem = vlist[(int)(t - (long long)z * M2)];
    const long long v = (long long)z * v2 + rem;
    const int j = rem / g.nx, i = rem - j * g.nx;

    double xi[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        xi[p] = th_in[(size_t)p * nvox + v];
        if (OPT && ((o.fixmask >> p) & 1)) xi[p] = o.lo[p];  // a fixed parameter sits at its value
    }
    // Q13: in-volume, in-mask 6-neighbourhood of the previous iterate (Jacobi); NQ = 10 (S8(f)2): the four in-plane
    // diagonals of the 3x3 clique as well
    const double delta[4] = {o.delta[0], OPT ? o.delta[1] : o.delta[0], OPT ? o.delta[2] : o.delta[0], OPT ? o.delta[3] : o.delta[0]};
    const int nq = o.nq;
    double nb[NQ][4];
    int nn = 0;
    {
        const int di[10] = {-1, 1, 0, 0, 0, 0, -1, 1, -1, 1}, dj[10] = {0, 0, -1, 1, 0, 0, -1, -1, 1, 1},
                  dz[10] = {0, 0, 0, 0, -1, 1, 0, 0, 0, 0};
        const int zr = z % g.nzr;  // slice index inside its replica
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int ii = i + di[q], jj = j + dj[q], zz = z + dz[q];
            // in-volume, in the same replica (slices [k nzr, (k+1) nzr)), in-mask
            const bool zok = dz[q] == 0 || (dz[q] < 0 ? zr > 0 : zr < g.nzr - 1);
            const bool ok = (!OPT || q < nq) && ii >= 0 && ii < g.nx && jj >= 0 && jj < g.ny && zok && mask[jj * g.nx + ii];
            if (ok) {
                const size_t w = (size_t)zz * v2 + (size_t)jj * g.nx + ii;
#pragma unroll
                for (int p = 0; p < 4; ++p) nb[nn][p] = th_in[(size_t)p * nvox + w];
                ++nn;
            }
        }
    }
    const XAddr xa = x_addr(g, (size_t)nvox, v, x_inner, Tp);

    double ev[15];
    if (FIRST) {
        lm_eval<WLS>(kin, fr, x, xa.base, xa.fstride, xi[0], xi[1], xi[2], xi[3], o.fixmask, ev);
        if (!LAST) {
#pragma unroll
            for (int q = 0; q < 15; ++q) st[(size_t)q * nfit + t] = ev[q];  // kept if this step is rejected
        }
    } else {
#pragma unroll
        for (int q = 0; q < 15; ++q) ev[q] = st[(size_t)q * nfit + t];
    }
    double gr[4] = {ev[10], ev[11], ev[12], ev[13]}, phi_old = ev[14];
    double curv[4] = {0.0, 0.0, 0.0, 0.0};  // OPT: Gauss-Newton curvature of the Huber sum, gamma sum_k H''
    for (int q = 0; q < nn; ++q)
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const double tt = xi[p] - nb[q][p];
            phi_old += gamma * huber(tt, delta[p]);
            gr[p] -= gamma * huber_d(tt, delta[p]);
            if (OPT && o.curv && fabs(tt) <= delta[p]) curv[p] += gamma;
        }

    double lam = lam_in[v];
    if (!(lam > 0.0)) lam = 1e-3 * fmax(fmax(ev[0], ev[2]), fmax(ev[5], ev[9]));  // Q15 first use
    double M[10];
#pragma unroll
    for (int q = 0; q < 10; ++q) M[q] = ev[q];
    M[0] += lam; M[2] += lam; M[5] += lam; M[9] += lam;
    if (OPT) { M[0] += curv[0]; M[2] += curv[1]; M[5] += curv[2]; M[9] += curv[3]; }
    double d[4];
    double phi = phi_old;
    if (!chol4(M, gr, d)) {
        lam = fmin(10.0 * lam, 1e30);  // not positive definite: treated as a rejected step
    } else {
        const double lo[4] = {0.0, 1e-4, 0.0, 0.0}, hi[4] = {2.0, 2.0, 1.0, 1.0};  // Q16
        double xt[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) xt[p] = fmin(fmax(xi[p] + d[p], OPT ? o.lo[p] : lo[p]), OPT ? o.hi[p] : hi[p]);
        lm_eval<WLS>(kin, fr, x, xa.base, xa.fstride, xt[0], xt[1], xt[2], xt[3], o.fixmask, ev);
        double phi_new = ev[14];
        for (int q = 0; q < nn; ++q)
#pragma unroll
            for (int p = 0; p < 4; ++p) phi_new += gamma * huber(xt[p] - nb[q][p], delta[p]);
        if (phi_new <= phi_old * (1.0 + 1e-6)) {  // Q15a: relative slack, see DESIGN.md section 3
#pragma unroll
            for (int p = 0; p < 4; ++p) xi[p] = xt[p];
            lam = fmax(lam / 10.0, 1e-30);
            phi = phi_new;
            if (!LAST) {
#pragma unroll
                for (int q = 0; q < 15; ++q) st[(size_t)q * nfit + t] = ev[q];
            }
        } else {
            lam = fmin(10.0 * lam, 1e30);
        }
    }
#pragma unroll
    for (int p = 0; p < 4; ++p) th_out[(size_t)p * nvox + v] = (TO)xi[p];
    lam_out[v] = (TO)lam;
    if (cost) cost[v] = (float)phi;
}

// K_i = K1 k3 / (k2 + k3)
__global__ void k_ki_map(const float *__restrict__ theta, float *__restrict__ ki, long long nvox) {
    const long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvox) return;
    const float K1 = theta[v], k2 = theta[nvox + v], k3 = theta[2 * nvox + v];
    const float a = k2 + k3;
    ki[v] = a > 0.f ? K1 * k3 / a : 0.f;
}

}  // namespace

int kcs_launch_ki_map(kcs_ctx *c, const float *theta, float *ki) {
    const long long nvox = (long long)c->n_vox;
    ProfScope ps(c, KCS_K_OTHER);
    k_ki_map<<<(unsigned)((nvox + 255) / 256), 256, 0, c->stream>>>(theta, ki, nvox);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

int kcs_launch_kinetic(kcs_ctx *c, const float *theta, float *F, float *J, int inner, int Tp, int z0, int nzc) {
    const long long nvox = (long long)c->n_vox;
    const size_t smem = sizeof(KFrame) * c->kin.T;
    if (nzc < 0) nzc = c->g.nz - z0;
    ProfScope ps(c, KCS_K_KINETIC);
    if (inner && !J) {
        const long long t0 = (long long)c->n_inmask2 * z0, nfit = (long long)c->n_inmask2 * nzc;
        if (nfit > 0)
            k_kinetic_inner<<<(unsigned)((nfit + 127) / 128), 128, smem, c->stream>>>(c->g, c->kin, theta, F, nvox, c->d_vlist, c->n_inmask2, Tp,
                                                                                      t0, t0 + nfit);
    } else
        k_kinetic<<<(unsigned)((nvox + 127) / 128), 128, smem, c->stream>>>(c->g, c->kin, theta, F, J, nvox, inner, Tp);
    LAUNCH_CHECK(c);
    return KCS_OK;
}

// in_f64 / out_f64: 0 = fp32 buffers (the caller's), 1 = the context's fp64 ping-pong buffers.
int kcs_launch_lm_step(kcs_ctx *c, const float *x, int x_inner, int Tp, const void *theta_in, int in_f64, void *theta_out,
                       int out_f64, const void *lam_in, void *lam_out, float gamma, float delta, float *cost, int z0, int nzc) {
    const long long nvox = (long long)c->n_vox;
    const size_t smem = sizeof(KFrame) * c->kin.T;
    const long long nfit = (long long)c->n_inmask2 * c->g.nz;  // stride of the carried sums: always the whole volume
    if (nzc < 0) nzc = c->g.nz - z0;
    const long long t0 = (long long)c->n_inmask2 * z0, t1 = t0 + (long long)c->n_inmask2 * nzc;
    if (t1 == t0) return KCS_OK;
    const unsigned grid = (unsigned)((t1 - t0 + KCS_LM_TPB - 1) / KCS_LM_TPB);
    ProfScope ps(c, KCS_K_LM);
    LmOpt o;
    o.fixmask = 0;
    for (int p = 0; p < 4; ++p) {
        o.delta[p] = c->has_delta4 ? c->delta4[p] : (double)delta;
        o.lo[p] = c->box_lo[p];
        o.hi[p] = c->box_hi[p];
        if (o.lo[p] == o.hi[p]) o.fixmask |= 1 << p;
    }
    o.nq = c->nbr_mode;
    o.curv = c->prior_curv ? 1 : 0;
    const bool opt = c->weighted || c->has_delta4 || c->nbr_mode != 6 || c->prior_curv || c->custom_box;
#define KCS_LM_GO2(TI, TO, OPT)                                                                                        \
    k_lm_step<TI, TO, OPT><<<grid, KCS_LM_TPB, smem, c->stream>>>(c->g, c->kin, x, x_inner, Tp, (const TI *)theta_in, (TO *)theta_out, \
                                                       (const TI *)lam_in, (TO *)lam_out, c->d_mask, c->d_vlist, c->n_inmask2, nvox, (double)gamma,  \
                                                       o, cost, c->lm_state, nfit, t0, t1)
#define KCS_LM_GO(TI, TO) do { if (opt) KCS_LM_GO2(TI, TO, true); else KCS_LM_GO2(TI, TO, false); } while (0)
    if (!in_f64 && !out_f64) KCS_LM_GO(float, float);
    else if (!in_f64 && out_f64) KCS_LM_GO(float, double);
    else if (in_f64 && out_f64) KCS_LM_GO(double, double);
    else KCS_LM_GO(double, float);
#undef KCS_LM_GO
#undef KCS_LM_GO2
    LAUNCH_CHECK(c);
    return KCS_OK;
}
